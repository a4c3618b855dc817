"""ChunkStream (copy / compute overlap over consecutive chunks) returns, chunk by chunk, what spd_search_host returns."""
import dataclasses

import numpy as np
import pytest
import torch

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1611_09704_b200 import build as B
    B.ensure_built()
    import paper_1611_09704_b200 as P
    P.lib()
    return P


@pytest.mark.parametrize("mode,nmax", [("sqrt", 32), ("linear", 16)])
def test_chunk_stream_equals_search_host(P, mode, nmax):
    from paper_1611_09704_b200.stream import ChunkStream
    base = gen.get_config(1)
    cap = 4096
    chunks = [torch.from_numpy(gen.make_array(dataclasses.replace(base, cid=base.cid + 100 * k))).pin_memory() for k in range(5)]
    cs = ChunkStream(base.n_dm, base.n_t, nmax, mode, base.threshold, capacity=cap, depth=2)
    got = cs.run(chunks)
    arena = torch.empty(P.search_host_arena_bytes(base.n_dm, base.n_t, nmax, cap), dtype=torch.uint8, device="cuda")
    h_out = torch.zeros((cap, 4), dtype=torch.int32).pin_memory()
    h_cnt = torch.zeros(1, dtype=torch.int64).pin_memory()
    counts = []
    for k, h in enumerate(chunks):
        total = P.spd_search_host(h, nmax, mode, base.threshold, h_out, h_cnt, None, arena)
        want = np.sort(h_out[:total].numpy().view(P.CAND_DTYPE).reshape(-1), order=["dm", "t"])
        rec, total2 = got[k]
        assert total2 == total and np.sort(rec, order=["dm", "t"]).tobytes() == want.tobytes()
        counts.append(total)
    assert len(set(counts)) > 1 and min(counts) > 0        # the chunks differ, and every one has detections


@pytest.mark.parametrize("mode,nmax", [("sqrt", 32), ("sqrt", 100), ("anchored", 64)])
def test_time_axis_chunks_with_overlap_equal_the_oracle_on_the_whole_series(P, mode, nmax):
    """Consecutive chunks along TIME overlap by Nmax - 1 (stream.time_chunks); with the statistics of the whole series the
    union of their records must be the ORACLE's candidate list of the concatenated series: every start sample searched
    exactly once, with every width (reading A9)."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    from paper_1611_09704_b200.stream import ChunkStream, time_chunks
    n_dm, n_t, k = 3, 4096, 4
    T = n_t + k * (n_t - nmax + 1)
    rng = np.random.Generator(np.random.PCG64(900 + nmax))
    x = (2.0 + 1.5 * rng.standard_normal((n_dm, T))).astype(np.float32)
    for c in range(1, k + 1):                              # pulses straddling every chunk boundary, and one at the very end
        b = c * (n_t - nmax + 1)
        x[c % n_dm, b - nmax // 2:b + nmax // 3] += 1.5
    x[0, T - 20:] += 4.0
    thr = 5.0
    o = O.search(x, nmax, mode, thr)
    st = o["stats"]
    assert [p[:2] for p in time_chunks(T, n_t, nmax)][:2] == [(0, n_t), (n_t - nmax + 1, n_t)]
    d_st = P.write_stats(st.mean, st.sigma, st.sigma_nmax, st.nmax_of_sigma)
    cs = ChunkStream(n_dm, n_t, nmax, mode, thr, capacity=1 << 16, depth=2)
    rec, total = cs.run_time_axis(torch.from_numpy(x).pin_memory(), d_st)
    r = CMP.compare_candidates(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 1 << 16, o["snr"], o["width"], o["margin"], thr,
                               x, st.mean, o["sig"])
    assert r, str(r)
    assert r.info["oracle_hits"] > 50 and (rec["t"] >= T - 20).any()


def test_chunk_stream_records_against_the_oracle(P):
    """ChunkStream output chunk by chunk against oracle.search (not against another CUDA call)."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    from paper_1611_09704_b200.stream import ChunkStream
    base = gen.get_config(1)
    chunks_np = [gen.make_array(dataclasses.replace(base, cid=base.cid + 100 * k)) for k in range(3)]
    cs = ChunkStream(base.n_dm, base.n_t, 32, "sqrt", base.threshold, capacity=4096, depth=2)
    got = cs.run([torch.from_numpy(c).pin_memory() for c in chunks_np])
    for c, (rec, total) in zip(chunks_np, got):
        o = O.search(c, 32, "sqrt", base.threshold)
        r = CMP.compare_candidates(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 4096, o["snr"], o["width"], o["margin"],
                                   base.threshold, c, o["stats"].mean, o["sig"])
        assert r, str(r)


def test_chunk_stream_refuses_to_overrun_its_slots(P):
    from paper_1611_09704_b200.stream import ChunkStream
    cs = ChunkStream(4, 2048, 8, "sqrt", 5.0, capacity=64, depth=1)
    h = torch.zeros((4, 2048), dtype=torch.float32).pin_memory()
    h[0, 5] = 1.0
    t = cs.submit(h)
    with pytest.raises(P.SpdError):
        cs.submit(h)
    rec, total, st = cs.result(t)
    assert int(st["n"][0]) == 4 * 2048
    with pytest.raises(P.SpdError):
        cs.result(t)


def test_chunk_stream_with_the_decimated_search_equals_the_oracle(P):
    """ChunkStream(decimated=(16, 3)): every chunk's list is the ORACLE's decimated candidate list (O5 + O4) of that chunk."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    from paper_1611_09704_b200.stream import ChunkStream
    base = gen.get_config(1)
    chunks = [gen.make_array(dataclasses.replace(base, cid=base.cid + 100 * k)) for k in range(3)]
    cs = ChunkStream(base.n_dm, base.n_t, 64, "sqrt", base.threshold, capacity=1 << 14, depth=2, decimated=(16, 3))
    got = cs.run([torch.from_numpy(c).pin_memory() for c in chunks])
    for x, (rec, total) in zip(chunks, got):
        o = O.search_decimated(x, 16, 3, "sqrt", base.threshold)
        r = CMP.compare_candidates_decimated(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 1 << 14, o["levels"], 16, base.threshold,
                                             x, o["stats"].mean, o["sig"])
        assert r and total > 0, str(r)
    with pytest.raises(P.SpdError):
        ChunkStream(base.n_dm, base.n_t, 100, "sqrt", base.threshold, decimated=(16, 3))      # nmax != w0 * 2^(levels-1)


def test_chunk_stream_result_raises_on_statistics_of_another_nmax(P):
    """LINEAR-mode statistics measured for another Nmax leave sigma_N undefined: the search writes the UINT64_MAX sentinel
    instead of a count (include/spd.h), and result() / run_time_axis must raise instead of handing back stale records."""
    from paper_1611_09704_b200.stream import ChunkStream
    n_dm, n_t, nmax = 4, 4096, 32
    rng = np.random.Generator(np.random.PCG64(77))
    x = torch.from_numpy(rng.standard_normal((n_dm, n_t)).astype(np.float32)).pin_memory()
    wrong = P.write_stats(0.0, 1.0, 4.0, 16)                 # sigma_Nmax of Nmax 16, searched with Nmax 32
    for dec in (None, (16, 2)):
        cs = ChunkStream(n_dm, n_t, nmax, "linear", 5.0, capacity=256, depth=2, decimated=dec)
        t = cs.submit(x, stats=wrong)
        with pytest.raises(P.SpdError, match="sigma_N is undefined"):
            cs.result(t)
        with pytest.raises(P.SpdError, match="sigma_N is undefined"):
            cs.run_time_axis(x, wrong)
        right = P.write_stats(0.0, 1.0, float(np.sqrt(nmax)), nmax)
        rec, total, _ = cs.result(cs.submit(x, stats=right))       # the stream is usable afterwards
        assert total >= 0 and rec.size == min(total, 256)


@pytest.mark.parametrize("mode,w0,levels", [("sqrt", 16, 3), ("anchored", 16, 4), ("sqrt", 32, 2)])
def test_time_axis_chunks_of_a_decimated_stream_equal_the_oracle_on_the_whole_series(P, mode, w0, levels):
    """run_time_axis on ChunkStream(decimated=...): chunk starts are multiples of 2^(levels-1), so each chunk's level grids
    are the series' own and the union of the records is the ORACLE's decimated candidate list of the concatenated series
    (reading A20)."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    from paper_1611_09704_b200.stream import ChunkStream, time_chunks
    nmax = w0 << (levels - 1)
    n_dm, n_t, k = 3, 4096, 3
    G = 1 << (levels - 1)
    step = (n_t - nmax + 1) // G * G
    assert step != n_t - nmax + 1                           # the unaligned step would shift the level grids
    T = n_t + k * step
    rng = np.random.Generator(np.random.PCG64(950 + nmax))
    x = (2.0 + 1.5 * rng.standard_normal((n_dm, T))).astype(np.float32)
    for c in range(1, k + 1):                               # pulses straddling every chunk boundary, and one at the very end
        b = c * step
        x[c % n_dm, b - nmax // 2:b + nmax // 3] += 1.5
    x[0, T - 20:] += 4.0
    thr = 5.0
    o = O.search_decimated(x, w0, levels, mode, thr)
    st = o["stats"]
    plan = time_chunks(T, n_t, nmax, G)
    assert all(s % G == 0 and length == n_t for s, length, _ in plan) and len(plan) == k + 1
    d_st = P.write_stats(st.mean, st.sigma, st.sigma_nmax, st.nmax_of_sigma)
    cs = ChunkStream(n_dm, n_t, nmax, mode, thr, capacity=1 << 16, depth=2, decimated=(w0, levels))
    rec, total = cs.run_time_axis(torch.from_numpy(x).pin_memory(), d_st)
    r = CMP.compare_candidates_decimated(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 1 << 16, o["levels"], w0, thr,
                                         x, st.mean, o["sig"])
    assert r and total > 50, str(r)
    assert (rec["t"] >= T - 20).any() and (rec["width"] > w0).any()


def test_chunk_stream_strided_and_pageable_sources_and_long_lists(P):
    """A time slice of a longer pinned series (row-strided) and a pageable tensor go through the slot's pinned staging buffer;
    a list longer than the SPEC_RECORDS copied with the count comes back whole through the count-sized second copy.  All
    three must give the records of the contiguous pinned chunk, byte for byte, and bytes_d2h must be what was moved."""
    from paper_1611_09704_b200 import stream as S
    n_dm, n_t, nmax, cap = 8, 8192, 16, 1 << 15
    rng = np.random.Generator(np.random.PCG64(4242))
    series = torch.from_numpy(rng.standard_normal((n_dm, 3 * n_t)).astype(np.float32)).pin_memory()
    view = series[:, n_t // 2:n_t // 2 + n_t]
    assert not view.is_contiguous()
    srcs = {"pinned": view.contiguous().pin_memory(), "strided": view, "pageable": view.contiguous()}
    assert srcs["pinned"].is_pinned() and not srcs["pageable"].is_pinned()
    for thr, long_list in ((4.5, False), (1.5, True)):
        got = {}
        for name, h in srcs.items():
            cs = S.ChunkStream(n_dm, n_t, nmax, "sqrt", thr, capacity=cap, depth=2)
            res = cs.run([h, h, h])                            # slot reuse: the staging buffer is rewritten while the pipeline runs
            assert all(r[1] == res[0][1] for r in res)
            rec, total = res[-1]
            assert total <= cap and rec.size == total
            assert (total > S.SPEC_RECORDS) == long_list
            assert cs.bytes_d2h == 8 + P.STATS_DTYPE.itemsize + 16 * max(total, S.SPEC_RECORDS)
            got[name] = np.sort(rec, order=["dm", "t"]).tobytes()
        d = srcs["pinned"].cuda()
        out, cnt = P.spd_search_fused(d, P.spd_stats(d), nmax, "sqrt", thr, capacity=cap)
        want, total = P.read_candidates(out, cnt)
        assert got["pinned"] == np.sort(want, order=["dm", "t"]).tobytes()
        assert got["strided"] == got["pinned"] and got["pageable"] == got["pinned"]


@pytest.mark.parametrize("mode,w0,levels,thr", [("sqrt", 16, 3, 6.0), ("linear", 16, 2, 4.0), ("sqrt", 32, 2, 2.5)])
def test_search_host_decimated_equals_the_oracle(P, mode, w0, levels, thr):
    """spd_search_host_decimated (host buffers in, host records out) against the ORACLE's decimated candidate list, and its
    statistics against the oracle's; the last case has a list longer than the 4096 records that travel with the count."""
    from oracle import spd_oracle as O
    from oracle import compare as CMP
    cfg = gen.get_config(1)
    x = gen.make_array(cfg)
    cap = 1 << 16
    h_x = torch.from_numpy(x).pin_memory()
    h_out = torch.zeros((cap, 4), dtype=torch.int32).pin_memory()
    h_count = torch.zeros(1, dtype=torch.int64).pin_memory()
    h_stats = torch.zeros(P.STATS_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    arena = torch.empty(P.search_host_decimated_arena_bytes(cfg.n_dm, cfg.n_t, w0, levels, cap), dtype=torch.uint8, device="cuda")
    total = P.spd_search_host_decimated(h_x, w0, levels, mode, thr, h_out, h_count, h_stats, arena)
    rec = h_out[:min(total, cap)].numpy().view(P.CAND_DTYPE).reshape(-1)
    o = O.search_decimated(x, w0, levels, mode, thr)
    g = h_stats.numpy().view(P.STATS_DTYPE)[0]
    r = CMP.compare_stats(float(g["mean"]), float(g["sigma"]), o["stats"], float(g["sigma_nmax"]) if mode != "sqrt" else None)
    assert r, str(r)
    r = CMP.compare_candidates_decimated(rec["dm"], rec["t"], rec["snr"], rec["width"], total, cap, o["levels"], w0, thr,
                                         x, o["stats"].mean, o["sig"])
    assert r and total > 0, str(r)
    if thr < 3.0:
        assert total > 4096
    with pytest.raises(P.SpdError):
        P.spd_search_host_decimated(h_x, w0, levels, mode, thr, h_out, h_count, h_stats, arena[:1024])
