"""Helpers of the -m gpu parity tests: run the CUDA path through the C-ABI binding, hand back numpy arrays."""
import numpy as np
import torch

import paper_1611_09704_b200 as P


def to_dev(x: np.ndarray, row_stride=None) -> torch.Tensor:
    """float32 [n_dm][n_t] -> CUDA tensor, optionally with a padded row stride (elements)."""
    n_dm, n_t = x.shape
    if row_stride is None or row_stride == n_t:
        return torch.from_numpy(np.ascontiguousarray(x)).cuda()
    buf = torch.full((n_dm, row_stride), float("nan"), dtype=torch.float32, device="cuda")
    buf[:, :n_t] = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return buf[:, :n_t]


def gpu_stats(x: np.ndarray, nmax_for_sigma=0, row_stride=None):
    d = to_dev(x, row_stride)
    st = P.spd_stats(d, nmax_for_sigma)
    return P.read_stats(st)[0], st


def gpu_sweep(x: np.ndarray, stats_dev: torch.Tensor, nmax: int, mode="sqrt", row_stride=None, want_width=True):
    d = to_dev(x, row_stride)
    snr, width = P.spd_boxcar_snr(d, stats_dev, nmax, mode, want_width=want_width)
    torch.cuda.synchronize()
    return snr.cpu().numpy(), (width.cpu().numpy() if width is not None else None), (d, snr, width)


def gpu_candidates(snr_dev, width_dev, thr, capacity=1 << 16):
    out, cnt = P.spd_candidates(snr_dev, width_dev, thr, capacity=capacity)
    rec, total = P.read_candidates(out, cnt)
    return rec, total


def gpu_fused(x_dev, stats_dev, nmax, mode, thr, capacity=1 << 16):
    out, cnt = P.spd_search_fused(x_dev, stats_dev, nmax, mode, thr, capacity=capacity)
    rec, total = P.read_candidates(out, cnt)
    return rec, total
