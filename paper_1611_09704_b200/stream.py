"""Chunked streaming with copy / compute overlap (the real-time pipeline shape of PAPER.md:97).

A telescope back-end produces one de-dispersed chunk [n_dm][n_t] after another.  `ChunkStream` keeps `depth` device
slots; the host-to-device copy of chunk i+1 runs on a copy stream while spd_stats + spd_search_fused (or, on request,
spd_search_fused_decimated) of chunk i run on a compute stream, and the statistics, the hit count and the records of a
finished chunk come back through pinned host buffers: the count, the statistics and the first SPEC_RECORDS records (64 KiB)
right behind the search, the rest of the list, if there is more, in one count-sized copy when the result is collected.
Only a contiguous pinned chunk is copied straight from where it lies; any other source (a time slice of a longer pinned
series, pageable memory) first goes through the slot's own pinned staging buffer, one host memcpy, so that the
host-to-device copy stays asynchronous and keeps overlapping the previous chunk's search.  This module is plumbing only (CUDA streams and events from PyTorch, argument marshalling); every step of
the search runs in the kernels behind the C ABI.

Chunks along TIME for the same DM trials must overlap by Nmax - 1 samples: the last Nmax - 1 samples of a row see only
the widths that fit (reading A9), so the next chunk starts Nmax - 1 samples before the end of this one and the
records of those last Nmax - 1 start samples are dropped from every chunk but the last (`time_chunks`,
`ChunkStream.run_time_axis`): every start sample of the series is then searched exactly once with every width.
With the decimated search the chunk starts must also be multiples of 2^(levels-1), or the pair sums of a later chunk
would straddle the pairs of the series' own decimation: `time_chunks(..., align=2^(levels-1))` rounds the step down
(the overlap grows by up to 2^(levels-1) - 1 samples) and the union of the records is then the decimated search of the
whole series, level grid for level grid.
"""
from __future__ import annotations

from typing import List, Optional, Tuple

import numpy as np
import torch

from . import binding as B


def time_chunks(n_total: int, chunk_len: int, nmax: int, align: int = 1) -> List[Tuple[int, int, int]]:
    """Cut a time axis of n_total samples into chunks of <= chunk_len samples that overlap by at least nmax - 1:
    [(start, length, keep)]; records with local start sample t < keep belong to the chunk (all of them in the last one).
    Every start is a multiple of `align` (2^(levels-1) for the decimated search; 1 for the exhaustive one)."""
    if not (1 <= nmax <= chunk_len and n_total >= 1 and align >= 1):
        raise ValueError("time_chunks: need 1 <= nmax <= chunk_len, n_total >= 1 and align >= 1")
    out, s, step = [], 0, (chunk_len - (nmax - 1)) // align * align
    if step < 1:
        raise ValueError("time_chunks: chunk_len - nmax + 1 is shorter than one aligned step")
    while True:
        length = min(chunk_len, n_total - s)
        last = s + length >= n_total
        out.append((s, length, length if last else step))
        if last:
            return out
        s += step


SPEC_RECORDS = 4096      # records copied back with the count, before the host knows how many there are (64 KiB)


class ChunkStream:
    def __init__(self, n_dm: int, n_t: int, nmax: int, mode="sqrt", threshold: float = 6.0, capacity: int = 1 << 20,
                 depth: int = 2, device="cuda", decimated: Optional[Tuple[int, int]] = None):
        """decimated = (w0, levels): search every chunk with spd_search_fused_decimated (nmax must equal
        w0 * 2^(levels-1)) instead of the exhaustive spd_search_fused."""
        if depth < 1:
            raise ValueError("depth >= 1")
        B.lib()
        self.decimated = None
        if decimated is not None:
            w0, levels = int(decimated[0]), int(decimated[1])
            if nmax != w0 << (levels - 1) or int(B.lib().spd_decimated_workspace_bytes(n_dm, n_t, w0, levels)) == 0:
                raise B.SpdError("ChunkStream: decimated = (w0, levels) needs w0 in {16, 32}, nmax == w0 * 2^(levels-1) <= 4096")
            self.decimated = (w0, levels)
        self.n_dm, self.n_t, self.nmax, self.mode, self.threshold, self.capacity = n_dm, n_t, int(nmax), mode, float(threshold), int(capacity)
        self.dev = torch.device(device)
        self.copy_stream = torch.cuda.Stream(self.dev)
        self.compute_stream = torch.cuda.Stream(self.dev)
        self.fetch_stream = torch.cuda.Stream(self.dev)       # remainder of a long list: must not queue behind the next chunk's search
        self.nsig = self.nmax if B._MODES[mode] != 0 else 0
        self.slots = []
        for _ in range(depth):
            out, cnt = B.new_candidates(self.capacity, self.dev)
            self.slots.append({
                "x": torch.empty((n_dm, n_t), dtype=torch.float32, device=self.dev),
                "stats": B.new_stats(self.dev), "ws": B.new_workspace(n_dm, n_t, self.nmax, self.dev),
                "dws": None if self.decimated is None else torch.empty(
                    int(B.lib().spd_decimated_workspace_bytes(n_dm, n_t, *self.decimated)), dtype=torch.uint8, device=self.dev),
                "out": out, "cnt": cnt,
                "h_out": torch.zeros((self.capacity, 4), dtype=torch.int32).pin_memory(),
                "h_cnt": torch.zeros(1, dtype=torch.int64).pin_memory(),
                "h_stats": torch.zeros(B.STATS_BYTES, dtype=torch.uint8).pin_memory(),
                "h_x": None,                                       # pinned staging buffer, made on first need
                "copied": torch.cuda.Event(), "done": torch.cuda.Event(), "busy": False,
            })
        self.next_slot = 0
        self.bytes_h2d = n_dm * n_t * 4
        self.spec = min(self.capacity, SPEC_RECORDS)
        self.bytes_d2h = 0                                     # device-to-host bytes moved for the chunk collected last

    def submit(self, h_x: torch.Tensor, stats: Optional[torch.Tensor] = None) -> int:
        """Enqueue one chunk (a CPU float32 [n_dm][n_t] tensor with unit time stride); returns a ticket.  A contiguous
        pinned tensor is copied asynchronously as it is; a row-strided or pageable one is first copied (on the host, now)
        into the slot's pinned staging buffer.  The slot's previous result must have been collected.  `stats`: a device
        spd_stats_t to search with (e.g. the statistics of a longer stretch of data) instead of measuring them on this
        chunk."""
        if h_x.is_cuda or h_x.dtype != torch.float32 or tuple(h_x.shape) != (self.n_dm, self.n_t) or h_x.stride(1) != 1:
            raise B.SpdError("h_x must be a CPU float32 [n_dm][n_t] tensor of the stream's shape with unit time stride")
        k = self.next_slot
        s = self.slots[k]
        if s["busy"]:
            raise B.SpdError("ChunkStream: collect the result of the oldest chunk before submitting another")
        self.next_slot = (k + 1) % len(self.slots)
        if not (h_x.is_contiguous() and h_x.is_pinned()):
            # torch would gather a strided source into a pageable temporary and copy that synchronously; the slot is free
            # (its last result was collected), so its staging buffer is no longer being read by an earlier copy
            if s["h_x"] is None:
                s["h_x"] = torch.empty((self.n_dm, self.n_t), dtype=torch.float32).pin_memory()
            s["h_x"].copy_(h_x)
            h_x = s["h_x"]
        with torch.cuda.stream(self.copy_stream):
            s["x"].copy_(h_x, non_blocking=True)
            s["copied"].record(self.copy_stream)
        with torch.cuda.stream(self.compute_stream):
            self.compute_stream.wait_event(s["copied"])
            if stats is None:
                B.spd_stats(s["x"], self.nsig, s["stats"], s["ws"], stream=self.compute_stream)
            else:
                s["stats"].copy_(stats, non_blocking=True)
            if self.decimated is None:
                B.spd_search_fused(s["x"], s["stats"], self.nmax, self.mode, self.threshold, s["out"], s["cnt"], ws=s["ws"],
                                   stream=self.compute_stream)
            else:
                B.spd_search_fused_decimated(s["x"], s["stats"], self.decimated[0], self.decimated[1], self.mode, self.threshold,
                                             s["out"], s["cnt"], ws=s["dws"], stream=self.compute_stream)
            s["h_cnt"].copy_(s["cnt"], non_blocking=True)
            s["h_stats"].copy_(s["stats"], non_blocking=True)
            s["h_out"][:self.spec].copy_(s["out"][:self.spec], non_blocking=True)   # the count is not known on the host yet
            s["done"].record(self.compute_stream)
        s["busy"] = True
        return k

    def result(self, ticket: int) -> Tuple[np.ndarray, int, np.ndarray]:
        """Wait for a chunk: (records written, total hit count, statistics).  The arrays are views of the slot's pinned
        buffers and are overwritten when the slot is reused."""
        s = self.slots[ticket]
        if not s["busy"]:
            raise B.SpdError("ChunkStream: no chunk in flight in this slot")
        s["done"].synchronize()
        s["busy"] = False
        total = B.check_count(int(s["h_cnt"][0]))      # raises on the 'sigma_N undefined' sentinel (stats of another Nmax)
        got = min(total, self.capacity)
        self.bytes_d2h = 8 + B.STATS_BYTES + 16 * self.spec
        if got > self.spec:                                    # a long list: the remainder in one copy of exactly its size
            with torch.cuda.stream(self.fetch_stream):         # the chunk is done (event above), so no ordering is needed
                s["h_out"][self.spec:got].copy_(s["out"][self.spec:got], non_blocking=True)
            self.fetch_stream.synchronize()
            self.bytes_d2h += 16 * (got - self.spec)
        rec = s["h_out"][:got].numpy().view(B.CAND_DTYPE).reshape(-1)
        return rec, total, s["h_stats"].numpy().view(B.STATS_DTYPE)

    def run_time_axis(self, h_series: torch.Tensor, stats: Optional[torch.Tensor] = None) -> Tuple[np.ndarray, int]:
        """Search a long series [n_dm][T] (pinned CPU tensor) as consecutive chunks of the stream's n_t samples that
        overlap by nmax - 1; returns (records with t in samples of the SERIES, number of records).  The last chunk must
        have the stream's length too: T = n_t + k step, step = n_t - nmax + 1 (decimated stream: rounded down to a
        multiple of 2^(levels-1) so that every chunk's level grids are the series' own; the result is then the
        decimated search of the whole series)."""
        T = h_series.shape[1]
        align = 1 if self.decimated is None else 1 << (self.decimated[1] - 1)
        plan = time_chunks(T, self.n_t, self.nmax, align)
        if any(length != self.n_t for _, length, _ in plan):
            raise B.SpdError(f"run_time_axis: the series length must be n_t + k * {(self.n_t - self.nmax + 1) // align * align}")
        recs: List[np.ndarray] = []
        tickets: List[Tuple[int, int, int]] = []

        def collect():
            tk, start, keep = tickets.pop(0)
            rec, total, _ = self.result(tk)
            if total > self.capacity:
                raise B.SpdError("run_time_axis: candidate buffer overflow")
            r = rec[rec["t"] < keep].copy()
            r["t"] += np.uint32(start)
            recs.append(r)
        for start, length, keep in plan:
            if len(tickets) == len(self.slots):
                collect()
            tickets.append((self.submit(h_series[:, start:start + length], stats), start, keep))
        while tickets:
            collect()
        out = np.concatenate(recs) if recs else np.zeros(0, dtype=B.CAND_DTYPE)
        return out, int(out.size)

    def run(self, chunks: List[torch.Tensor]) -> List[Tuple[np.ndarray, int]]:
        """Convenience: push a list of chunks through the pipeline in order; returns copies of (records, count)."""
        res: List[Optional[Tuple[np.ndarray, int]]] = []
        tickets: List[int] = []
        for h in chunks:
            if len(tickets) == len(self.slots):
                rec, total, _ = self.result(tickets.pop(0))
                res.append((rec.copy(), total))
            tickets.append(self.submit(h))
        for t in tickets:
            rec, total, _ = self.result(t)
            res.append((rec.copy(), total))
        return res
