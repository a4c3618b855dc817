#!/usr/bin/env python
"""bench.py -- throughput of the single-pulse-detection hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--nmax M] [--impl ours|reference]

One "step" = one pass of the whole hot path (spd_stats -> spd_boxcar_snr -> spd_candidates) over one chunk of
synthetic de-dispersed data (gen/, config C; default 3 = the SKA-like chunk BASELINE.json's metric and target
are quoted on).  Prints ONE JSON line on rank 0.  Inputs are resident in HBM for `value`; `e2e` goes through
spd_search_host with pinned HOST buffers (H2D + D2H inside the timed region).
`--impl reference` times the CPU oracle (oracle/) on a bounded row sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "DM×time samples/s through boxcar SNR search (×real-time); HBM GB/s vs peak"
SM_COUNT, FP32_LANES_PER_SM = 148, 128
# Sweep roofline: every (sample, width) pair needs one fp32 add and one fp32 multiply = 2 FMA-pipe
# lane-ops; peak = 148 SMs x 128 lanes x sm_max_mhz.  `roofline.frac` uses exactly that.  The instruction set cannot reach
# it: the measured cost of the loop's own mix is 2.5 issue slots per pair (add, multiply, half a 3-input maximum; packed
# FADD2 / FMUL2 take two slots: profiles/r02_fp32_issue_rates.md), reported beside it as `frac_of_issue_slot_floor`.
FMA_OPS_PER_PAIR = 2.0
ISSUE_SLOTS_PER_PAIR = 2.5
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_dram_traffic.csv")   # kernel,config,nmax,n_dm,dram_read_bytes,dram_write_bytes,source


def ncu_traffic(kernel: str, config: int, nmax: int, n_dm: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch from a tracked `ncu --set full` capture of exactly this
    workload (profiles/ncu_dram_traffic.csv); None when there is no capture for it."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    import csv
    for row in csv.DictReader(open(TRAFFIC_CSV)):
        if (row["kernel"] == kernel and int(row["config"]) == config and int(row["nmax"]) == nmax and int(row["n_dm"]) == n_dm):
            return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), row["source"]
    return None, None


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows[-3:]]
        for r in rows:
            f = [s.strip() for s in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def pick_workload(args):
    cfg = gen.get_config(args.config)
    nmax = args.nmax or (128 if cfg.cid == 5 else cfg.nmax[0])
    n_dm = args.rows or cfg.n_dm
    return cfg, nmax, n_dm


def workload_name(cfg, nmax, n_dm):
    return f"{cfg.name}: {n_dm} DM trials x {cfg.n_t} samples f32, Nmax={nmax}, sigma_N {cfg.sigma_mode}, threshold {cfg.threshold}"


def oracle_sample_rate(cfg, nmax, target_s: float, rank_seed: int = 0):
    """The oracle, as it stands, on a bounded row sample of the workload: (samples/s, cores, sample text, seconds)."""
    from oracle import spd_oracle as O
    O.build()
    cores = O.num_threads()
    rows = min(cfg.n_dm, max(2, cores))
    x = gen.make_rows(cfg, list(range(rows)))
    t0 = time.time()
    O.search(x, nmax, cfg.sigma_mode, cfg.threshold)
    dt = time.time() - t0
    want = int(min(cfg.n_dm, max(rows, rows * target_s / max(dt, 1e-3))))
    want = max(cores, want - want % cores) if want >= cores else want
    if want > rows:
        x = gen.make_array(cfg, row_lo=0, row_hi=want)
        t0 = time.time()
        O.search(x, nmax, cfg.sigma_mode, cfg.threshold)
        dt = time.time() - t0
        rows = want
    n = rows * cfg.n_t
    # per-core figure: the sweep alone, one thread, a 4-row subset
    x4 = gen.make_rows(cfg, list(range(min(4, cfg.n_dm))))
    st4 = O.full_stats(x4, nmax if cfg.sigma_mode != "sqrt" else 0)
    sig4 = O.sigma_table(st4.sigma, st4.sigma_nmax, nmax, cfg.sigma_mode)
    prev = os.environ.get("OMP_NUM_THREADS")
    O.set_num_threads(1)
    t0 = time.time()
    O.sweep(x4, st4.mean, sig4)
    dt1 = time.time() - t0
    O.set_num_threads(cores)
    extra = {"ns_per_pair": dt * 1e9 / (n * nmax), "threads": cores,
             "one_thread": {"rows": int(x4.shape[0]), "seconds": dt1, "ns_per_pair": dt1 * 1e9 / (x4.size * nmax),
                            "what": "oracle sweep (O3) alone, 1 OpenMP thread"}}
    return n / dt, cores, f"first {rows} of {cfg.n_dm} rows ({n} samples, {dt:.1f} s of oracle time: stats+sweep+candidates)", dt, extra


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import spd_oracle as O
    O.build()
    cfg, nmax, n_dm = pick_workload(args)
    cores = O.num_threads()
    rows = min(n_dm, max(2, 2 * cores))
    x = gen.make_rows(cfg, list(range(rows)))
    for _ in range(min(args.warmup, 1)):
        O.search(x, nmax, cfg.sigma_mode, cfg.threshold)
    t0 = time.time()
    for _ in range(args.steps):
        O.search(x, nmax, cfg.sigma_mode, cfg.threshold)
    dt = (time.time() - t0) / args.steps
    n = rows * cfg.n_t
    v = n / dt
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": "samples/s", "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(cfg, nmax, n_dm), "sample": f"each step = first {rows} rows ({n} samples)"},
           "cpu_baseline": {"value": v, "unit": "samples/s", "cores": cores, "kind": "oracle",
                            "sample": f"first {rows} of {n_dm} rows per step, {args.steps} steps"},
           "e2e": {"value": v, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def extra_legs(torch, P, args, dev, step, barrier, d_x, h_x, st, ws, out, cnt, arena, n_dm, n_t, nmax, nmax_sigma, mode, thr, cap):
    """The legs beside the headline step: CUDA-graph replay, fused search, e2e through spd_search_host, ChunkStream pipeline."""
    # ---- the same step captured once in a CUDA graph and replayed (matters for launch-latency-bound shapes such as config 1) ----
    gs = torch.cuda.Stream(dev)
    with torch.cuda.stream(gs):
        step()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=gs):
            step()
    torch.cuda.synchronize()
    q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    graph.replay()
    q0.record()
    for _ in range(args.steps):
        graph.replay()
    q1.record()
    torch.cuda.synchronize()
    graph_ms = q0.elapsed_time(q1) / args.steps
    del graph

    # ---- the fused search (spd_stats + spd_search_fused: planes never written), timed beside the plane path ---------------
    g0, g1, g2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    fsteps = max(1, min(args.steps, 5))
    P.spd_stats(d_x, nmax_sigma, st, ws); P.spd_search_fused(d_x, st, nmax, mode, thr, out, cnt, ws=ws)
    torch.cuda.synchronize()
    g0.record()
    for _ in range(fsteps):
        P.spd_stats(d_x, nmax_sigma, st, ws)
    g1.record()
    for _ in range(fsteps):
        P.spd_search_fused(d_x, st, nmax, mode, thr, out, cnt, ws=ws)
    g2.record()
    torch.cuda.synchronize()
    fused_ms = (g0.elapsed_time(g1) + g1.elapsed_time(g2)) / fsteps
    fused_kernel_ms = g1.elapsed_time(g2) / fsteps
    hits_fused = int(cnt.item())

    # ---- end to end through the C ABI with HOST buffers (H2D of x, D2H of stats + count + list each step) ------
    h_out = torch.zeros((cap, 4), dtype=torch.int32).pin_memory()
    h_cnt = torch.zeros(1, dtype=torch.int64).pin_memory()
    h_st = torch.zeros(P.STATS_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(1):
        P.spd_search_host(h_x, nmax, mode, thr, h_out, h_cnt, h_st, arena)
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(e2e_steps):
        hits_e2e = P.spd_search_host(h_x, nmax, mode, thr, h_out, h_cnt, h_st, arena)
    f1.record()
    barrier()
    ms_e2e = f0.elapsed_time(f1) / e2e_steps

    # ---- the same chunk through the copy / compute pipeline (ChunkStream): H2D of chunk i+1 overlaps the search of chunk i ----
    from paper_1611_09704_b200.stream import ChunkStream
    cs = ChunkStream(n_dm, n_t, nmax, mode, thr, capacity=cap, depth=2, device=dev)
    pipe_steps = max(4, e2e_steps)
    cs.run([h_x, h_x])                                  # warm-up
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    pipe_res = cs.run([h_x] * pipe_steps)
    p1.record()
    barrier()
    ms_pipe = p0.elapsed_time(p1) / pipe_steps
    hits_pipe = pipe_res[-1][1]
    d2h_pipe = cs.bytes_d2h                             # what the last chunk actually moved back (count + stats + records)
    del cs

    return graph_ms, fused_ms, fused_kernel_ms, hits_fused, ms_e2e, hits_e2e, e2e_steps, ms_pipe, hits_pipe, pipe_steps, d2h_pipe


def decimated_leg(torch, P, args, d_x, st, ws, n_dm, n_t, nmax, nmax_sigma, mode, thr, cap, hbm_peak):
    """spd_stats + spd_boxcar_snr_decimated + spd_candidates_decimated (reading A20) for the same Nmax as
    w0 = 16 x levels; an approximation of the exhaustive step (sensitivity >= sqrt(0.9)), reported beside it."""
    if nmax < 32 or nmax % 16 or (nmax // 16) & (nmax // 16 - 1):
        return None
    w0, levels = 16, (nmax // 16).bit_length()
    stride = P.decimated_level_offset(n_t, levels)
    snr = torch.empty((n_dm, stride), dtype=torch.float32, device=d_x.device)
    wid = torch.empty((n_dm, stride), dtype=torch.uint16, device=d_x.device)
    dws = torch.empty(int(P.lib().spd_decimated_workspace_bytes(n_dm, n_t, w0, levels)), dtype=torch.uint8, device=d_x.device)
    out, cnt = P.new_candidates(cap, d_x.device)

    def run():
        P.spd_stats(d_x, nmax_sigma, st, ws)
        P.spd_boxcar_snr_decimated(d_x, st, w0, levels, mode, snr, wid, dws)
        P.spd_candidates_decimated(snr, wid, n_t, levels, thr, out, cnt)
    for _ in range(2):
        run()
    torch.cuda.synchronize()
    steps = max(1, min(args.steps, 5))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        run()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    hits_planes = int(cnt.item())

    def run_fused():
        P.spd_stats(d_x, nmax_sigma, st, ws)
        P.spd_search_fused_decimated(d_x, st, w0, levels, mode, thr, out, cnt, ws=dws)
    for _ in range(2):
        run_fused()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        run_fused()
    e1.record()
    torch.cuda.synchronize()
    ms_fused = e0.elapsed_time(e1) / steps
    hits_fused = int(cnt.item())
    n = n_dm * n_t
    frac_sum = sum(0.5 ** l for l in range(levels))
    # fused: x read by the statistics and by level 0; level l >= 1 reads its series and level l < L-1 writes the next one
    alg_fused = n * (4 + 4 + 4 * (frac_sum - 1) + 4 * sum(0.5 ** l for l in range(1, levels)))
    # bytes that must cross HBM: x read once by the statistics and once by the search, planes of every level written once and
    # their SNR read once by the candidate selection; the decimated series are intermediates (credit: none)
    alg_bytes = n * (4 + 4 + (4 + 2 + 4) * frac_sum)
    fused = {"ms_per_step": ms_fused, "hits": hits_fused, "value": n / (ms_fused * 1e-3), "unit": "samples/s per GPU",
             "algorithmic_bytes_per_sample": alg_fused / n, "hbm_GBps": alg_fused / (ms_fused * 1e-3) / 1e9,
             "hbm_frac_of_measured": alg_fused / (ms_fused * 1e-3) / 1e9 / hbm_peak,
             "note": "spd_stats + spd_search_fused_decimated: the same list with the threshold in the level kernels, no planes"}
    return {"ms_per_step": ms, "w0": w0, "levels": levels, "hits": hits_planes, "value": n / (ms * 1e-3), "unit": "samples/s per GPU", "fused": fused,
            "algorithmic_bytes_per_sample": alg_bytes / n, "hbm_GBps": alg_bytes / (ms * 1e-3) / 1e9,
            "hbm_frac_of_measured": alg_bytes / (ms * 1e-3) / 1e9 / hbm_peak,
            "note": "spd_stats + spd_boxcar_snr_decimated + spd_candidates_decimated: widths 1..16, then 18..32 step 2, 36..64 step 4, ...; "
                    "an approximation (worst-case sensitivity sqrt(0.9) of the exhaustive search), not the headline step"}


def run_ours(args):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    from paper_1611_09704_b200 import build as _build
    _build.ensure_built()                      # a fresh clone has no libspd.so (git-ignored); nvcc is in the image
    import paper_1611_09704_b200 as P
    P.lib()

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; reporting n_gpus={world}", file=sys.stderr)
    torch.cuda.set_device(local)
    if world > 1 or args.shard == "rows":      # the sharded step all-gathers the statistics (also at world size 1)
        if "MASTER_ADDR" not in os.environ:
            import socket
            with socket.socket() as sk:
                sk.bind(("127.0.0.1", 0))
                os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(sk.getsockname()[1]), RANK="0", WORLD_SIZE="1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    cfg, nmax, n_dm = pick_workload(args)
    shard_rows = args.shard == "rows"
    row_lo = 0
    n_dm_total = n_dm
    if shard_rows:         # strong scaling: ONE chunk, DM rows cut across the ranks (shard.py; statistics exchanged by all-gather + eq. 2 fold)
        from paper_1611_09704_b200 import shard as S
        row_lo, row_hi = S.row_partition(n_dm_total, world, rank)
        n_dm = row_hi - row_lo
        if n_dm < 1:
            raise SystemExit("bench.py --shard rows: fewer DM rows than ranks")
    elif world > 1:        # weak scaling: every rank searches its own, differently seeded chunk of the same shape
        import dataclasses
        cfg = dataclasses.replace(cfg, cid=cfg.cid + 100 * rank)
    n_t, mode, thr = cfg.n_t, cfg.sigma_mode, cfg.threshold
    n = n_dm * n_t
    cap = 1 << 20

    # ---- synthetic input (host, pinned), then resident in HBM -----------------------------------------------
    t_gen = time.time()
    h_x = torch.empty((n_dm, n_t), dtype=torch.float32, pin_memory=True)
    gen.make_array(cfg, out=h_x.numpy(), threads=max(1, (os.cpu_count() or 1) // max(1, world)), row_lo=row_lo, row_hi=row_lo + n_dm)
    t_gen = time.time() - t_gen
    arena = torch.empty(P.search_host_arena_bytes(n_dm, n_t, nmax, cap), dtype=torch.uint8, device=dev)   # of the e2e leg
    d_x = torch.empty((n_dm, n_t), dtype=torch.float32, device=dev)
    d_snr = torch.empty((n_dm, n_t), dtype=torch.float32, device=dev)
    d_w = torch.empty((n_dm, n_t), dtype=torch.uint16, device=dev)
    d_x.copy_(h_x, non_blocking=True)
    st = P.new_stats(dev)
    ws = P.new_workspace(n_dm, n_t, nmax, dev)
    out, cnt = P.new_candidates(cap, dev)
    nmax_sigma = nmax if mode != "sqrt" else 0
    # our kernels per step: stats_partial[_win] + stats_finalize, [sigma_table_kernel unless eq. 4 with nmax % 8 == 0], sweep,
    # zero_count + candidates_compact (shard mode adds stats_merge_kernel)
    launches_per_step = 2 + (0 if (mode == "sqrt" and nmax % 8 == 0) else 1) + 1 + 2 + (1 if shard_rows else 0)

    def step(ev=None):
        if shard_rows:     # local Chan triples, all-gather of the 80-byte structs (NCCL), eq. 2 fold in rank order: whole-chunk mu, sigma
            st.copy_(S.sharded_stats(d_x, nmax_sigma, ws=ws))
        else:
            P.spd_stats(d_x, nmax_sigma, st, ws)
        if ev: ev[0].record()
        P.spd_boxcar_snr(d_x, st, nmax, mode, d_snr, d_w, ws)
        if ev: ev[1].record()
        P.spd_candidates(d_snr, d_w, thr, out, cnt)
        if ev: ev[2].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    w0 = time.time()
    e0.record()
    for i in range(args.steps):
        step(evs[i])
    e1.record()
    barrier()
    w1 = time.time()
    clocks = sampler.stop(w0, w1) if rank == 0 else None
    ms_total = e0.elapsed_time(e1)
    t_stats = [e0.elapsed_time(evs[0][0])] + [evs[i - 1][2].elapsed_time(evs[i][0]) for i in range(1, args.steps)]
    t_sweep = [evs[i][0].elapsed_time(evs[i][1]) for i in range(args.steps)]
    t_cand = [evs[i][1].elapsed_time(evs[i][2]) for i in range(args.steps)]
    hits = int(cnt.item())
    stats_host = P.read_stats(st)[0]

    extras = not shard_rows and not args.no_e2e
    graph_ms = fused_ms = fused_kernel_ms = ms_e2e = ms_pipe = float("nan")
    hits_fused = hits_e2e = hits_pipe = -1
    e2e_steps = pipe_steps = d2h_pipe = 0
    if shard_rows and not args.no_e2e:
        # end to end for the sharded run: H2D of the rank's rows from pinned memory, shard.sharded_search (fused), D2H of count + records
        h_out = torch.zeros((cap, 4), dtype=torch.int32).pin_memory()
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for it in range(e2e_steps + 1):
            if it == 1:
                barrier(); f0.record()
            d_x.copy_(h_x, non_blocking=True)
            o_, c_, _, _ = S.sharded_search(d_x, row_lo, nmax, mode, thr, cap)
            hits_e2e = int(c_.item())
            h_out[:min(hits_e2e, cap)].copy_(o_[:min(hits_e2e, cap)])
        f1.record(); barrier()
        ms_e2e = f0.elapsed_time(f1) / e2e_steps
    if extras:
        (graph_ms, fused_ms, fused_kernel_ms, hits_fused, ms_e2e, hits_e2e, e2e_steps, ms_pipe, hits_pipe, pipe_steps, d2h_pipe) = \
            extra_legs(torch, P, args, dev, step, barrier, d_x, h_x, st, ws, out, cnt, arena, n_dm, n_t, nmax, nmax_sigma, mode, thr, cap)
    del arena
    dec = None
    if extras:
        dec = decimated_leg(torch, P, args, d_x, st, ws, n_dm, n_t, nmax, nmax_sigma, mode, thr, cap, _peaks()[0])

    # ---- max over ranks -------------------------------------------------------------------------------------------
    t = torch.tensor([ms_total, ms_e2e], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total, ms_e2e = float(t[0]), float(t[1])
    ms_step = ms_total / args.steps

    if rank == 0:
        hbm_peak, sm_max_mhz, peak_kind = _peaks()
        pairs = float(n) * nmax
        sweep_ms = float(np.mean(t_sweep))
        # Roofline of the sweep, exactly as SURVEY.md 8(d) defines it: HBM side 10 B/sample (4 read + 4 snr + 2 width) against
        # the measured copy bandwidth; arithmetic side 2 FMA-pipe lane-ops per (sample, width) pair against 148 SMs x 128
        # lanes x sm_max_mhz.  Whichever floor is larger binds and gives `frac`.
        alu_peak = SM_COUNT * FP32_LANES_PER_SM * sm_max_mhz * 1e6 / 1e12          # T lane-ops/s
        alu_ach = FMA_OPS_PER_PAIR * pairs / (sweep_ms * 1e-3) / 1e12
        hbm_ach = 10.0 * n / (sweep_ms * 1e-3) / 1e9
        hbm_bound = (10.0 * n / (hbm_peak * 1e9)) > (FMA_OPS_PER_PAIR * pairs / (alu_peak * 1e12))
        roof = ({"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_ach / hbm_peak}
                if hbm_bound else
                {"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": alu_ach / alu_peak})
        sweep_kernel = "boxcar_snr_sweep_narrow" if nmax <= 32 else "boxcar_snr_sweep"
        traffic, traffic_src = ncu_traffic(sweep_kernel, args.config, nmax, n_dm)
        roof.update({"kernel": sweep_kernel, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": f"{peak_kind} (MEASURED_PEAKS.json)" if roof["bound"] == "hbm" else
                                    "derived (SURVEY.md 8(d), DESIGN.md section 7): 148 SM x 128 fp32 lanes x sm_max_mhz; 2 FMA-pipe lane-ops (add, multiply) per (sample,width) pair",
                     "ms_per_launch": sweep_ms, "algorithmic_bytes_per_sample": 10, "fma_ops_per_pair": FMA_OPS_PER_PAIR,
                     "hbm_GBps": hbm_ach, "hbm_frac_of_measured": hbm_ach / hbm_peak, "hbm_frac_of_8TBps": hbm_ach / 8000.0,
                     "alu_Tops": alu_ach, "alu_frac": alu_ach / alu_peak,
                     "frac_of_issue_slot_floor": ISSUE_SLOTS_PER_PAIR * pairs / (sweep_ms * 1e-3) / 1e12 / alu_peak,
                     "issue_slot_floor_note": "2.5 issue slots per pair (FADD2 + FMUL2 = 2 slots per lane pair, half an FMNMX3) is what the "
                                              "instruction set allows for add + multiply + running maximum: profiles/r02_fp32_issue_rates.md"})
        cpu = None
        if not args.no_cpu_baseline:
            v, cores, sample, _, extra = oracle_sample_rate(gen.get_config(args.config), nmax, args.cpu_seconds)
            cpu = {"value": v, "unit": "samples/s", "cores": cores, "kind": "oracle", "sample": sample}
            cpu.update(extra)
        n_job = n_dm_total * n_t if shard_rows else world * n          # samples all ranks processed per step
        value = n_job / (ms_step * 1e-3)
        nan_to_none = lambda v: None if (isinstance(v, float) and v != v) else v
        res = {
            "metric": METRIC, "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "strong" if shard_rows else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, nmax, n_dm_total if shard_rows else n_dm), "config_id": args.config,
                       "n_dm": n_dm_total if shard_rows else n_dm, "n_t": n_t,
                       "nmax": nmax, "sigma_mode": mode, "threshold": thr, "samples_per_step_per_gpu": n,
                       "l2": "input 4n bytes >> 126 MB L2, no flush needed" if n * 4 > (1 << 29) else "L2-resident input (small config)",
                       "parallelism": (f"one chunk, DM rows sharded over {world} GPU(s): local spd_stats, NCCL all-gather of the 80-byte "
                                       "spd_stats_t, eq. 2 fold in rank order, then sweep + candidates on the local rows") if shard_rows
                                      else f"independent chunks, one per GPU (x{world}), no data-path collective",
                       "gen_seconds": round(t_gen, 1)},
            "x_realtime": (n_t * cfg.t_samp) / (ms_step * 1e-3) if cfg.cid % 100 == 3 else None,
            "breakdown_ms": {"spd_stats": float(np.mean(t_stats)), "spd_boxcar_snr": sweep_ms, "spd_candidates": float(np.mean(t_cand))},
            "stats_GBps": 4.0 * n * (2 if nmax_sigma else 1) / (float(np.mean(t_stats)) * 1e-3) / 1e9,
            "candidates_GBps": 4.0 * n / (float(np.mean(t_cand)) * 1e-3) / 1e9,
            "cuda_graph": {"ms_per_step": nan_to_none(graph_ms), "note": "the same three calls captured once and replayed"},
            "fused_search": {"ms_per_step": nan_to_none(fused_ms), "spd_search_fused_ms": nan_to_none(fused_kernel_ms), "hits": hits_fused,
                             "value": nan_to_none(n / (fused_ms * 1e-3)), "unit": "samples/s per GPU",
                             "note": "spd_stats + spd_search_fused (same candidate list, SNR and width planes never written); not the headline step"},
            "decimated_search": dec,
            "hits": hits, "mean": float(stats_host["mean"]), "sigma": float(stats_host["sigma"]),
            "clocks": clocks,
            "e2e": {"value": nan_to_none(n_job / (ms_e2e * 1e-3)), "unit": "samples/s", "ms_per_step": nan_to_none(ms_e2e), "steps": e2e_steps,
                    "h2d_bytes_per_step": n * 4, "d2h_bytes_per_step": 8 + P.STATS_DTYPE.itemsize + 16 * max(0, min(hits_e2e, cap)),
                    "path": "fused",
                    "api": ("paper_1611_09704_b200.shard.sharded_search per rank (pinned host rows -> H2D, spd_stats, all-gather + spd_stats_merge, "
                            "spd_search_fused, D2H of count and records)") if shard_rows else
                           ("spd_search_host (pinned host buffers; H2D, spd_stats, spd_search_fused, D2H of statistics, count and records; "
                            "the SNR / width planes are never written on this path)")},
            "e2e_pipelined": {"value": nan_to_none(n / (ms_pipe * 1e-3)), "unit": "samples/s per GPU", "ms_per_step": nan_to_none(ms_pipe), "steps": pipe_steps,
                              "hits": hits_pipe, "h2d_bytes_per_step": n * 4, "d2h_bytes_per_step": d2h_pipe,
                              "api": "paper_1611_09704_b200.stream.ChunkStream (two slots: H2D of chunk i+1 overlaps spd_stats + spd_search_fused of chunk i)"},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roof,
            "cpu_baseline": cpu,
        }
        print(json.dumps(res), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE config 1..5 (default 3 = SKA-like)")
    ap.add_argument("--nmax", type=int, default=0, help="override the widest boxcar")
    ap.add_argument("--rows", type=int, default=0, help="override n_dm (smaller runs for profiling)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="only the headline step (short runs under ncu / compute-sanitizer)")
    ap.add_argument("--shard", default="none", choices=["none", "rows"],
                    help="rows: ONE chunk with its DM rows cut across the ranks (strong scaling, shard.py) instead of one chunk per rank")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU), exactly as the driver's torchrun line does
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
