"""DM-row sharding of ONE chunk across ranks ("on each of DM trial").

One process per GPU.  Rows are cut into contiguous blocks; the sweep and the candidate selection of a block need
nothing from the other blocks.  The statistics do: every rank computes the Chan triple (n, T, S) of its own rows with
`spd_stats`, the 80-byte `spd_stats_t` structs are ALL-GATHERED (the only exchange step of the path; eq. 2 is not a
plain sum, so it is an all-gather followed by a local fold, not an all-reduce) and every rank folds them in RANK ORDER
with eq. 2 (`spd_stats_merge`), which makes mu and sigma bit-identical on every rank.

This module only moves the structs (torch.distributed: NCCL on GPUs, gloo in the CPU tests) and calls the C ABI; it
computes nothing itself.  Candidate records carry the LOCAL row index; `row_lo` is returned beside them (the global
DM index is the same caller-side affine map as the physical DM of include/spd.h).
"""
from __future__ import annotations

from typing import Optional, Tuple

import torch
import torch.distributed as dist

from . import binding as B


def row_partition(n_dm: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced row block [lo, hi) of `rank`: the first n_dm % world ranks hold one row more."""
    if not (n_dm >= 0 and world >= 1 and 0 <= rank < world):
        raise ValueError("row_partition: need n_dm >= 0, world >= 1, 0 <= rank < world")
    q, r = divmod(n_dm, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def gather_stats(stats_local: torch.Tensor, group=None) -> torch.Tensor:
    """All-gather one spd_stats_t (uint8[80]) per rank -> uint8[world * 80] in rank order, on the input's device."""
    if stats_local.dtype != torch.uint8 or stats_local.numel() != B.STATS_BYTES:
        raise ValueError("gather_stats: expected one spd_stats_t as uint8[%d]" % B.STATS_BYTES)
    world = dist.get_world_size(group)
    out = torch.empty(world * B.STATS_BYTES, dtype=torch.uint8, device=stats_local.device)
    dist.all_gather_into_tensor(out, stats_local.contiguous(), group=group)
    return out


def sharded_stats(x_local: torch.Tensor, nmax_for_sigma: int = 0, group=None, ws: Optional[torch.Tensor] = None) -> torch.Tensor:
    """spd_stats on this rank's rows, all-gather, eq. 2 fold in rank order: the statistics of the WHOLE chunk.
    A rank that holds no rows contributes an all-zero struct (n = 0), which eq. 2 skips."""
    if x_local.shape[0] > 0:
        st = B.spd_stats(x_local, nmax_for_sigma, ws=ws)
    else:
        st = B.new_stats(x_local.device)
    parts = gather_stats(st, group)
    return B.spd_stats_merge(parts, dist.get_world_size(group))


def sharded_search(x_local: torch.Tensor, row_lo: int, nmax: int, mode, threshold: float, capacity: int,
                   group=None, fused: bool = True):
    """The whole path on this rank's row block with whole-chunk statistics.
    Returns (records uint8 tensor, count tensor, row_lo, stats): global dm = row_lo + record.dm."""
    nsig = nmax if B._MODES[mode] != 0 else 0
    st = sharded_stats(x_local, nsig, group)
    if x_local.shape[0] == 0:
        out, cnt = B.new_candidates(capacity, x_local.device)
        return out, cnt, row_lo, st
    if fused:
        out, cnt = B.spd_search_fused(x_local, st, nmax, mode, threshold, capacity=capacity)
    else:
        snr, width = B.spd_boxcar_snr(x_local, st, nmax, mode)
        out, cnt = B.spd_candidates(snr, width, threshold, capacity=capacity)
    return out, cnt, row_lo, st
