"""DM-row sharding on the GPU: the two row blocks of a 2-rank run, emulated as one process over
both blocks' data (B200_PROFILING.md: never run ranks that wait on one another on one GPU), and the real
torch.distributed code path at world_size 1 over NCCL."""
import os
import socket

import numpy as np
import pytest
import torch

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1611_09704_b200 as P
    from paper_1611_09704_b200 import build as B
    B.ensure_built()
    P.lib()
    return P


def _unsharded(P, x, nmax, mode, thr):
    d = torch.from_numpy(x).cuda()
    st = P.spd_stats(d, nmax if mode != "sqrt" else 0)
    out, cnt = P.spd_search_fused(d, st, nmax, mode, thr, capacity=1 << 16)
    rec, total = P.read_candidates(out, cnt)
    return st, np.sort(rec, order=["dm", "t"]), total


@pytest.mark.parametrize("mode,nmax", [("sqrt", 32), ("linear", 40)])
def test_two_row_blocks_merged_equal_the_whole_chunk(P, mode, nmax):
    from paper_1611_09704_b200 import shard as S
    cfg = gen.get_config(1)
    x = gen.make_array(cfg)
    st_all, rec_all, total_all = _unsharded(P, x, nmax, mode, cfg.threshold)
    parts, blocks = [], []
    for rank in range(2):
        lo, hi = S.row_partition(cfg.n_dm, 2, rank)
        d = torch.from_numpy(np.ascontiguousarray(x[lo:hi])).cuda()
        parts.append(P.spd_stats(d, nmax if mode != "sqrt" else 0))
        blocks.append((lo, d))
    st = P.spd_stats_merge(torch.cat(parts), 2)
    a, b = P.read_stats(st)[0], P.read_stats(st_all)[0]
    assert a["n"] == b["n"] and a["n_b"] == b["n_b"]
    for k in ("mean", "sigma") + (("sigma_nmax",) if mode != "sqrt" else ()):
        assert abs(a[k] - b[k]) <= 1e-7 * max(abs(b[k]), b["sigma"])      # fp32 warp chunks are shifted by a per-call K: not bit-equal
    recs = []
    for lo, d in blocks:
        out, cnt = P.spd_search_fused(d, st_all, nmax, mode, cfg.threshold, capacity=1 << 16)   # same statistics => identical records
        r, _ = P.read_candidates(out, cnt)
        r = r.copy()
        r["dm"] += lo
        recs.append(r)
    got = np.sort(np.concatenate(recs), order=["dm", "t"])
    assert got.tobytes() == rec_all.tobytes() and total_all > 0


@pytest.mark.parametrize("mode,nmax,world", [("sqrt", 32, 2), ("linear", 40, 3), ("sqrt", 64, 5)])
def test_row_blocks_against_the_oracle(P, mode, nmax, world):
    """The sharded path against oracle.search of the WHOLE chunk (not against another CUDA call): per-block spd_stats, eq. 2
    fold of the gathered structs in rank order (spd_stats_merge), sweep + threshold per block with the merged statistics,
    records concatenated with their row offsets.  world = 5 > some blocks' share exercises uneven and (for n_dm = 4) empty blocks."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    from paper_1611_09704_b200 import shard as S
    n_dm = 64 if world < 5 else 4
    cfg = gen.custom_config(n_dm, 8192, cid=55, mu=10.0, sigma=3.0)
    x = gen.make_rows(cfg, list(range(n_dm)))
    x[1, 4000:4030] += 12.0                            # 4 sigma per sample: well above the threshold also under eq. 5
    thr = 5.0
    o = O.search(x, nmax, mode, thr)
    nsig = nmax if mode != "sqrt" else 0
    parts, blocks = [], []
    for rank in range(world):
        lo, hi = S.row_partition(n_dm, world, rank)
        if hi > lo:
            d = torch.from_numpy(np.ascontiguousarray(x[lo:hi])).cuda()
            parts.append(P.spd_stats(d, nsig))
            blocks.append((lo, d))
        else:
            parts.append(P.new_stats("cuda"))          # a rank without rows contributes an all-zero struct
    st = P.spd_stats_merge(torch.cat(parts), world)
    g = P.read_stats(st)[0]
    r = CMP.compare_stats(float(g["mean"]), float(g["sigma"]), o["stats"], float(g["sigma_nmax"]) if nsig else None)
    assert r, str(r)
    recs = []
    for lo, d in blocks:
        out, cnt = P.spd_search_fused(d, st, nmax, mode, thr, capacity=1 << 16)
        rr, _ = P.read_candidates(out, cnt)
        rr = rr.copy()
        rr["dm"] += lo
        recs.append(rr)
    rec = np.concatenate(recs)
    # the oracle planes were made with the ORACLE's statistics, the GPU records with the merged GPU statistics (1e-6 apart)
    rc = CMP.compare_candidates(rec["dm"], rec["t"], rec["snr"], rec["width"], rec.size, 1 << 16, o["snr"], o["width"], o["margin"], thr,
                                x, o["stats"].mean, o["sig"])
    assert rc, str(rc)
    assert rc.info["oracle_hits"] > 10


def test_sharded_search_world1_nccl(P):
    import torch.distributed as dist
    from paper_1611_09704_b200 import shard as S
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        cfg = gen.get_config(1)
        x = gen.make_array(cfg)
        st_all, rec_all, total_all = _unsharded(P, x, 32, "sqrt", cfg.threshold)
        lo, hi = S.row_partition(cfg.n_dm, 1, 0)
        out, cnt, row_lo, st = S.sharded_search(torch.from_numpy(x[lo:hi]).cuda(), lo, 32, "sqrt", cfg.threshold, 1 << 16)
        rec, total = P.read_candidates(out, cnt)
        assert row_lo == 0 and total == total_all
        assert np.sort(rec, order=["dm", "t"]).tobytes() == rec_all.tobytes()
        a, b = P.read_stats(st)[0], P.read_stats(st_all)[0]
        assert a["mean"] == b["mean"] and a["sigma"] == b["sigma"]
    finally:
        dist.destroy_process_group()
