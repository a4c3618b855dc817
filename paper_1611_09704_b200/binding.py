"""Thin ctypes binding of libspd.so (include/spd.h): argument marshalling only.

PyTorch supplies device memory and streams; every step of the path runs in the CUDA kernels of
csrc/.  There is no CPU fallback: a missing library or a non-CUDA tensor raises.
Function names mirror the C ABI (spd_stats, spd_boxcar_snr, spd_candidates, ...).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspd.so")

SPD_SIGMA_SQRT, SPD_SIGMA_LINEAR, SPD_SIGMA_LINEAR_ANCHORED = 0, 1, 2
_MODES = {"sqrt": 0, "linear": 1, "anchored": 2, 0: 0, 1: 1, 2: 2}

STATS_DTYPE = np.dtype([("mean", "<f8"), ("sigma", "<f8"), ("sigma_nmax", "<f8"), ("T", "<f8"), ("S", "<f8"),
                        ("T_b", "<f8"), ("S_b", "<f8"), ("n", "<u8"), ("n_b", "<u8"),
                        ("nmax_of_sigma", "<i4"), ("_pad", "<i4")])
CAND_DTYPE = np.dtype([("dm", "<u4"), ("t", "<u4"), ("snr", "<f4"), ("width", "<u4")])
STATS_BYTES = STATS_DTYPE.itemsize      # 80
assert CAND_DTYPE.itemsize == 16


class SpdError(RuntimeError):
    pass


_lib = None


def lib() -> C.CDLL:
    """Load libspd.so (built in-tree by paper_1611_09704_b200.build); fail loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise SpdError(f"{LIB_PATH} not found: build it with `python -m paper_1611_09704_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        i64, i32, vp, f32, u64, sz = C.c_int64, C.c_int, C.c_void_p, C.c_float, C.c_uint64, C.c_size_t
        L.spd_status_string.argtypes = [i32]; L.spd_status_string.restype = C.c_char_p
        L.spd_workspace_bytes.argtypes = [i64, i64, i32]; L.spd_workspace_bytes.restype = sz
        L.spd_stats.argtypes = [vp, i64, i64, i64, i32, vp, vp, sz, vp]
        L.spd_stats_merge.argtypes = [vp, i32, vp, vp]
        L.spd_boxcar_snr.argtypes = [vp, i64, i64, i64, vp, i32, i32, vp, vp, vp, sz, vp]
        L.spd_candidates.argtypes = [vp, vp, i64, i64, i64, f32, vp, u64, vp, vp]
        L.spd_search_fused.argtypes = [vp, i64, i64, i64, vp, i32, i32, f32, vp, u64, vp, vp, sz, vp]
        L.spd_search_host_arena_bytes.argtypes = [i64, i64, i32, u64]; L.spd_search_host_arena_bytes.restype = sz
        L.spd_search_host.argtypes = [vp, i64, i64, i32, i32, f32, vp, u64, vp, vp, vp, sz, vp]
        L.spd_search_host_decimated_arena_bytes.argtypes = [i64, i64, i32, i32, u64]; L.spd_search_host_decimated_arena_bytes.restype = sz
        L.spd_search_host_decimated.argtypes = [vp, i64, i64, i32, i32, i32, f32, vp, u64, vp, vp, vp, sz, vp]
        L.spd_workspace_bytes_rows.argtypes = [i64, i64, i32]; L.spd_workspace_bytes_rows.restype = sz
        L.spd_stats_rows.argtypes = [vp, i64, i64, i64, i32, vp, vp, sz, vp]
        L.spd_stats_rows_noalloc.argtypes = [vp, i64, i64, i64, i32, vp, vp]
        L.spd_stats_rows_noalloc_max_rows.argtypes = []; L.spd_stats_rows_noalloc_max_rows.restype = i64
        L.spd_boxcar_snr_rows.argtypes = [vp, i64, i64, i64, vp, i32, i32, vp, vp, vp, sz, vp]
        L.spd_search_fused_rows.argtypes = [vp, i64, i64, i64, vp, i32, i32, f32, vp, u64, vp, vp, sz, vp]
        L.spd_decimated_level_offset.argtypes = [i64, i32]; L.spd_decimated_level_offset.restype = i64
        L.spd_decimated_workspace_bytes.argtypes = [i64, i64, i32, i32]; L.spd_decimated_workspace_bytes.restype = sz
        L.spd_boxcar_snr_decimated.argtypes = [vp, i64, i64, i64, vp, i32, i32, i32, vp, vp, i64, vp, sz, vp]
        L.spd_candidates_decimated.argtypes = [vp, vp, i64, i64, i64, i32, f32, vp, u64, vp, vp]
        L.spd_search_fused_decimated.argtypes = [vp, i64, i64, i64, vp, i32, i32, i32, f32, vp, u64, vp, vp, sz, vp]
        for f in ("spd_stats", "spd_stats_merge", "spd_boxcar_snr", "spd_candidates", "spd_search_fused", "spd_search_host",
                  "spd_boxcar_snr_decimated", "spd_candidates_decimated", "spd_search_fused_decimated", "spd_stats_rows", "spd_boxcar_snr_rows",
                  "spd_search_fused_rows", "spd_stats_rows_noalloc", "spd_search_host_decimated"):
            getattr(L, f).restype = i32
        _lib = L
    return _lib


def _check(code: int, what: str) -> None:
    if code != 0:
        raise SpdError(f"{what}: {lib().spd_status_string(code).decode()} ({code})")


def _stream(stream: Optional[torch.cuda.Stream]) -> int:
    return (stream or torch.cuda.current_stream()).cuda_stream


def _plane(x: torch.Tensor, dtype, name: str) -> Tuple[int, int, int]:
    if not (x.is_cuda and x.dtype == dtype and x.dim() == 2 and x.stride(1) == 1 and x.stride(0) >= x.shape[1]):
        raise SpdError(f"{name} must be a CUDA {dtype} [n_dm][n_t] tensor with unit time stride")
    return x.shape[0], x.shape[1], x.stride(0)


def workspace_bytes(n_dm: int, n_t: int, nmax: int) -> int:
    return int(lib().spd_workspace_bytes(n_dm, n_t, nmax))


def new_workspace(n_dm: int, n_t: int, nmax: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(256, workspace_bytes(n_dm, n_t, max(nmax, 1))), dtype=torch.uint8, device=device)


def new_stats(device="cuda", count: int = 1) -> torch.Tensor:
    return torch.zeros(count * STATS_BYTES, dtype=torch.uint8, device=device)


def read_stats(stats: torch.Tensor) -> np.ndarray:
    """Device spd_stats_t -> numpy structured array (synchronises)."""
    return stats.cpu().numpy().view(STATS_DTYPE)


def write_stats(mean: float, sigma: float, sigma_nmax: float = float("nan"), nmax_of_sigma: int = 0,
                device="cuda") -> torch.Tensor:
    """A caller-made spd_stats_t (e.g. mu = 0, sigma = 1 for tests), as the C header allows."""
    a = np.zeros(1, dtype=STATS_DTYPE)
    a["mean"], a["sigma"], a["sigma_nmax"], a["nmax_of_sigma"] = mean, sigma, sigma_nmax, nmax_of_sigma
    return torch.from_numpy(a.view(np.uint8).copy()).to(device)


def spd_stats(x: torch.Tensor, nmax_for_sigma: int = 0, stats: Optional[torch.Tensor] = None,
              ws: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    stats = new_stats(x.device) if stats is None else stats
    ws = new_workspace(n_dm, n_t, nmax_for_sigma, x.device) if ws is None else ws
    _check(lib().spd_stats(x.data_ptr(), n_dm, n_t, rs, int(nmax_for_sigma), stats.data_ptr(), ws.data_ptr(),
                           ws.numel(), _stream(stream)), "spd_stats")
    return stats


def spd_stats_merge(parts: torch.Tensor, count: int, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    out = new_stats(parts.device) if out is None else out
    _check(lib().spd_stats_merge(parts.data_ptr(), int(count), out.data_ptr(), _stream(stream)), "spd_stats_merge")
    return out


def spd_boxcar_snr(x: torch.Tensor, stats: torch.Tensor, nmax: int, mode="sqrt",
                   snr: Optional[torch.Tensor] = None, width: Optional[torch.Tensor] = None,
                   ws: Optional[torch.Tensor] = None, stream=None, want_width: bool = True):
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if snr is None:
        snr = torch.empty_strided((n_dm, n_t), (rs, 1), dtype=torch.float32, device=x.device)
    if width is None and want_width:
        width = torch.empty_strided((n_dm, n_t), (rs, 1), dtype=torch.uint16, device=x.device)
    if _plane(snr, torch.float32, "snr") != (n_dm, n_t, rs) or (width is not None and _plane(width, torch.uint16, "width") != (n_dm, n_t, rs)):
        raise SpdError("snr / width planes must share x's shape and row stride")
    ws = new_workspace(n_dm, n_t, nmax, x.device) if ws is None else ws
    _check(lib().spd_boxcar_snr(x.data_ptr(), n_dm, n_t, rs, stats.data_ptr(), int(nmax), _MODES[mode], snr.data_ptr(),
                                width.data_ptr() if width is not None else None, ws.data_ptr(), ws.numel(),
                                _stream(stream)), "spd_boxcar_snr")
    return snr, width


def new_candidates(capacity: int, device="cuda") -> Tuple[torch.Tensor, torch.Tensor]:
    return (torch.empty((max(1, capacity), 4), dtype=torch.int32, device=device),
            torch.zeros(1, dtype=torch.int64, device=device))


def spd_candidates(snr: torch.Tensor, width: torch.Tensor, threshold: float, out: Optional[torch.Tensor] = None,
                   count: Optional[torch.Tensor] = None, capacity: int = 1 << 20, stream=None):
    n_dm, n_t, rs = _plane(snr, torch.float32, "snr")
    if _plane(width, torch.uint16, "width") != (n_dm, n_t, rs):
        raise SpdError("width plane must share snr's shape and row stride")
    if out is None or count is None:
        out, count = new_candidates(capacity, snr.device)
    _check(lib().spd_candidates(snr.data_ptr(), width.data_ptr(), n_dm, n_t, rs, float(threshold), out.data_ptr(),
                                out.shape[0], count.data_ptr(), _stream(stream)), "spd_candidates")
    return out, count


def spd_search_fused(x: torch.Tensor, stats: torch.Tensor, nmax: int, mode, threshold: float,
                     out: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None,
                     capacity: int = 1 << 20, ws: Optional[torch.Tensor] = None, stream=None):
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if out is None or count is None:
        out, count = new_candidates(capacity, x.device)
    ws = new_workspace(n_dm, n_t, nmax, x.device) if ws is None else ws
    _check(lib().spd_search_fused(x.data_ptr(), n_dm, n_t, rs, stats.data_ptr(), int(nmax), _MODES[mode], float(threshold),
                                  out.data_ptr(), out.shape[0], count.data_ptr(), ws.data_ptr(), ws.numel(),
                                  _stream(stream)), "spd_search_fused")
    return out, count


def new_workspace_rows(n_dm: int, n_t: int, nmax: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(256, int(lib().spd_workspace_bytes_rows(n_dm, n_t, max(nmax, 1)))), dtype=torch.uint8, device=device)


def spd_stats_rows(x: torch.Tensor, nmax_for_sigma: int = 0, stats: Optional[torch.Tensor] = None,
                   ws: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """One spd_stats_t per DM row: uint8[n_dm * 80] on the device (read_stats gives the structured array)."""
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    stats = new_stats(x.device, n_dm) if stats is None else stats
    ws = new_workspace_rows(n_dm, n_t, nmax_for_sigma, x.device) if ws is None else ws
    _check(lib().spd_stats_rows(x.data_ptr(), n_dm, n_t, rs, int(nmax_for_sigma), stats.data_ptr(), ws.data_ptr(), ws.numel(),
                                _stream(stream)), "spd_stats_rows")
    return stats


def spd_stats_rows_noalloc(x: torch.Tensor, stats: torch.Tensor, nmax_for_sigma: int = 0, stream=None) -> torch.Tensor:
    """spd_stats_rows for code that may not allocate device memory: a stage inside a real-time pipeline whose host
    framework owns every byte of the card and hands the stage its input and output buffers, nothing else.

    `x` and `stats` (uint8[n_dm * 80], e.g. a slice of the framework's output buffer) are the caller's; the workspace
    that spd_stats_rows would need is a 3 MiB array inside libspd.so.  Neither this function nor the C call behind it
    allocates.  At most noalloc_max_rows() = 8192 rows per call: more raises SpdError (SPD_ERR_NOALLOC_LIMIT) and
    launches nothing.  Results equal spd_stats_rows bit for bit.  Calls share the array, so issue them on one stream
    (or order them with events): calls that overlap on the GPU corrupt each other's statistics.  Make the first call on
    each device during start-up; it resolves the array's device address."""
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if stats.device != x.device or stats.dtype != torch.uint8 or not stats.is_contiguous() or stats.numel() < n_dm * STATS_BYTES:
        raise SpdError("stats must be a contiguous uint8 tensor of n_dm * 80 bytes on x's device")
    _check(lib().spd_stats_rows_noalloc(x.data_ptr(), n_dm, n_t, rs, int(nmax_for_sigma), stats.data_ptr(), _stream(stream)),
           "spd_stats_rows_noalloc")
    return stats


def noalloc_max_rows() -> int:
    return int(lib().spd_stats_rows_noalloc_max_rows())


def spd_boxcar_snr_rows(x: torch.Tensor, stats_rows: torch.Tensor, nmax: int, mode="sqrt",
                        snr: Optional[torch.Tensor] = None, width: Optional[torch.Tensor] = None,
                        ws: Optional[torch.Tensor] = None, stream=None):
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if stats_rows.numel() != n_dm * STATS_BYTES:
        raise SpdError("stats_rows must hold one spd_stats_t per DM row")
    if snr is None:
        snr = torch.empty_strided((n_dm, n_t), (rs, 1), dtype=torch.float32, device=x.device)
    if width is None:
        width = torch.empty_strided((n_dm, n_t), (rs, 1), dtype=torch.uint16, device=x.device)
    ws = new_workspace_rows(n_dm, n_t, nmax, x.device) if ws is None else ws
    _check(lib().spd_boxcar_snr_rows(x.data_ptr(), n_dm, n_t, rs, stats_rows.data_ptr(), int(nmax), _MODES[mode], snr.data_ptr(),
                                     width.data_ptr(), ws.data_ptr(), ws.numel(), _stream(stream)), "spd_boxcar_snr_rows")
    return snr, width


def spd_search_fused_rows(x: torch.Tensor, stats_rows: torch.Tensor, nmax: int, mode, threshold: float,
                          out: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None,
                          capacity: int = 1 << 20, ws: Optional[torch.Tensor] = None, stream=None):
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if stats_rows.numel() != n_dm * STATS_BYTES:
        raise SpdError("stats_rows must hold one spd_stats_t per DM row")
    if out is None or count is None:
        out, count = new_candidates(capacity, x.device)
    ws = new_workspace_rows(n_dm, n_t, nmax, x.device) if ws is None else ws
    _check(lib().spd_search_fused_rows(x.data_ptr(), n_dm, n_t, rs, stats_rows.data_ptr(), int(nmax), _MODES[mode], float(threshold),
                                       out.data_ptr(), out.shape[0], count.data_ptr(), ws.data_ptr(), ws.numel(),
                                       _stream(stream)), "spd_search_fused_rows")
    return out, count


def decimated_level_offset(n_t: int, level: int) -> int:
    """First element of level `level` inside a row of the packed planes; level == levels gives the row length."""
    return int(lib().spd_decimated_level_offset(n_t, level))


def spd_boxcar_snr_decimated(x: torch.Tensor, stats: torch.Tensor, w0: int, levels: int, mode="sqrt",
                             snr: Optional[torch.Tensor] = None, width: Optional[torch.Tensor] = None,
                             ws: Optional[torch.Tensor] = None, stream=None):
    """Decimation in time + boxcar (include/spd.h): returns the packed (snr f32, width u16) planes [n_dm][plane_stride];
    level l of row d is [d, decimated_level_offset(n_t, l) : + (n_t >> l)]."""
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    stride = decimated_level_offset(n_t, levels)
    if stride < 0:
        raise SpdError("spd_boxcar_snr_decimated: invalid n_t / levels")
    if snr is None:
        snr = torch.empty((n_dm, stride), dtype=torch.float32, device=x.device)
    if width is None:
        width = torch.empty((n_dm, stride), dtype=torch.uint16, device=x.device)
    if _plane(snr, torch.float32, "snr") != _plane(width, torch.uint16, "width") or snr.shape[0] != n_dm:
        raise SpdError("packed snr / width planes must share one shape and row stride")
    need = int(lib().spd_decimated_workspace_bytes(n_dm, n_t, int(w0), int(levels)))
    if need == 0:
        raise SpdError("spd_boxcar_snr_decimated: w0 must be 16 or 32, 1 <= levels <= 8, w0 * 2^(levels-1) <= 4096")
    ws = torch.empty(need, dtype=torch.uint8, device=x.device) if ws is None else ws
    _check(lib().spd_boxcar_snr_decimated(x.data_ptr(), n_dm, n_t, rs, stats.data_ptr(), int(w0), int(levels), _MODES[mode],
                                          snr.data_ptr(), width.data_ptr(), snr.stride(0), ws.data_ptr(), ws.numel(),
                                          _stream(stream)), "spd_boxcar_snr_decimated")
    return snr, width


def spd_candidates_decimated(snr: torch.Tensor, width: torch.Tensor, n_t: int, levels: int, threshold: float,
                             out: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None,
                             capacity: int = 1 << 20, stream=None):
    n_dm, _, stride = _plane(snr, torch.float32, "snr")
    if out is None or count is None:
        out, count = new_candidates(capacity, snr.device)
    _check(lib().spd_candidates_decimated(snr.data_ptr(), width.data_ptr(), n_dm, int(n_t), stride, int(levels), float(threshold),
                                          out.data_ptr(), out.shape[0], count.data_ptr(), _stream(stream)), "spd_candidates_decimated")
    return out, count


def spd_search_fused_decimated(x: torch.Tensor, stats: torch.Tensor, w0: int, levels: int, mode, threshold: float,
                               out: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None,
                               capacity: int = 1 << 20, ws: Optional[torch.Tensor] = None, stream=None):
    """Decimated search with the threshold in the level kernels (include/spd.h): one list for all levels, no planes."""
    n_dm, n_t, rs = _plane(x, torch.float32, "x")
    if out is None or count is None:
        out, count = new_candidates(capacity, x.device)
    need = int(lib().spd_decimated_workspace_bytes(n_dm, n_t, int(w0), int(levels)))
    if need == 0:
        raise SpdError("spd_search_fused_decimated: w0 must be 16 or 32, 1 <= levels <= 8, w0 * 2^(levels-1) <= 4096")
    ws = torch.empty(need, dtype=torch.uint8, device=x.device) if ws is None else ws
    _check(lib().spd_search_fused_decimated(x.data_ptr(), n_dm, n_t, rs, stats.data_ptr(), int(w0), int(levels), _MODES[mode],
                                            float(threshold), out.data_ptr(), out.shape[0], count.data_ptr(), ws.data_ptr(),
                                            ws.numel(), _stream(stream)), "spd_search_fused_decimated")
    return out, count


def check_count(total: int) -> int:
    """The hit count as read into an int64: -1 is 0xFFFFFFFFFFFFFFFF, the 'sigma_N undefined' sentinel of spd_search_fused /
    spd_search_fused_decimated (include/spd.h): no record was written, so there is no list to hand back."""
    if total < 0:
        raise SpdError("spd_search_fused: sigma_N is undefined (a LINEAR mode fed statistics measured for another Nmax)")
    return total


def read_candidates(out: torch.Tensor, count: torch.Tensor) -> Tuple[np.ndarray, int]:
    """Device list -> (numpy structured array of the written records, total hit count).  Synchronises."""
    total = check_count(int(count.item()))
    got = min(total, out.shape[0])
    rec = out[:got].cpu().numpy().view(CAND_DTYPE).reshape(-1)
    return rec, total


def search_host_arena_bytes(n_dm: int, n_t: int, nmax: int, capacity: int) -> int:
    return int(lib().spd_search_host_arena_bytes(n_dm, n_t, nmax, capacity))


def spd_search_host(h_x: torch.Tensor, nmax: int, mode, threshold: float, h_out: torch.Tensor, h_count: torch.Tensor,
                    h_stats: Optional[torch.Tensor], arena: torch.Tensor, stream=None) -> int:
    """Whole path from HOST tensors (pinned for asynchronous copies); returns the hit count.  Synchronises."""
    if h_x.is_cuda or h_x.dtype != torch.float32 or h_x.dim() != 2 or not h_x.is_contiguous():
        raise SpdError("h_x must be a contiguous CPU float32 [n_dm][n_t] tensor")
    if h_out.is_cuda or h_out.dtype != torch.int32 or h_out.dim() != 2 or h_out.shape[1] != 4 or h_count.is_cuda:
        raise SpdError("h_out must be a CPU int32 [capacity][4] tensor, h_count a CPU int64 tensor")
    n_dm, n_t = h_x.shape
    _check(lib().spd_search_host(h_x.data_ptr(), n_dm, n_t, int(nmax), _MODES[mode], float(threshold), h_out.data_ptr(),
                                 h_out.shape[0], h_count.data_ptr(), h_stats.data_ptr() if h_stats is not None else None,
                                 arena.data_ptr(), arena.numel(), _stream(stream)), "spd_search_host")
    return check_count(int(h_count[0]))


def search_host_decimated_arena_bytes(n_dm: int, n_t: int, w0: int, levels: int, capacity: int) -> int:
    return int(lib().spd_search_host_decimated_arena_bytes(n_dm, n_t, w0, levels, capacity))


def spd_search_host_decimated(h_x: torch.Tensor, w0: int, levels: int, mode, threshold: float, h_out: torch.Tensor,
                              h_count: torch.Tensor, h_stats: Optional[torch.Tensor], arena: torch.Tensor, stream=None) -> int:
    """spd_search_host with the decimated search (Nmax = w0 * 2^(levels-1)); returns the hit count.  Synchronises."""
    if h_x.is_cuda or h_x.dtype != torch.float32 or h_x.dim() != 2 or not h_x.is_contiguous():
        raise SpdError("h_x must be a contiguous CPU float32 [n_dm][n_t] tensor")
    if h_out.is_cuda or h_out.dtype != torch.int32 or h_out.dim() != 2 or h_out.shape[1] != 4 or h_count.is_cuda:
        raise SpdError("h_out must be a CPU int32 [capacity][4] tensor, h_count a CPU int64 tensor")
    n_dm, n_t = h_x.shape
    _check(lib().spd_search_host_decimated(h_x.data_ptr(), n_dm, n_t, int(w0), int(levels), _MODES[mode], float(threshold),
                                           h_out.data_ptr(), h_out.shape[0], h_count.data_ptr(),
                                           h_stats.data_ptr() if h_stats is not None else None,
                                           arena.data_ptr(), arena.numel(), _stream(stream)), "spd_search_host_decimated")
    return check_count(int(h_count[0]))
