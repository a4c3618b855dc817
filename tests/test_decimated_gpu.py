"""-m gpu parity of the decimated search (spd_boxcar_snr_decimated / spd_candidates_decimated, reading A20)
against oracle O5, level by level and element by element, under the tolerances of DESIGN.md section 5."""
import math

import numpy as np
import pytest
import torch

import gen
from oracle import compare as CMP
from oracle import spd_oracle as O

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


def rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _run(P, x, w0, levels, mode="sqrt", stats=None, thr=None, stride=None):
    from gpu_util import to_dev
    nmax = w0 << (levels - 1)
    o = O.full_stats(x, nmax if mode != "sqrt" else 0) if stats is None else stats
    st = P.write_stats(o.mean, o.sigma, o.sigma_nmax, o.nmax_of_sigma)
    d = to_dev(x, stride)
    snr, width = P.spd_boxcar_snr_decimated(d, st, w0, levels, mode)
    lv = O.sweep_decimated(x, o.mean, o.sigma, o.sigma_nmax, mode, w0, levels)
    sig_all = O.sigma_table(o.sigma, o.sigma_nmax, nmax, mode)
    n_t = x.shape[1]
    g_snr, g_w = snr.cpu().numpy(), width.cpu().numpy()
    infos = []
    for L in lv:
        off, n_l = P.decimated_level_offset(n_t, L["level"]), n_t >> L["level"]
        r = CMP.compare_planes_level(x, o.mean, sig_all, w0, L, g_snr[:, off:off + n_l], g_w[:, off:off + n_l])
        assert r, f"level {L['level']}: {r}"
        infos.append(r.info)
    if thr is not None:
        out, cnt = P.spd_candidates_decimated(snr, width, n_t, levels, thr, capacity=1 << 20)
        rec, total = P.read_candidates(out, cnt)
        want = 0
        got = set(zip(rec["dm"].tolist(), rec["t"].tolist(), rec["width"].tolist()))
        assert len(got) == total                       # one record per (level position): (dm, t, width) is unique
        for L in lv:
            D, off, n_l = L["D"], P.decimated_level_offset(n_t, L["level"]), n_t >> L["level"]
            gs = g_snr[:, off:off + n_l]
            hit = np.argwhere(gs >= np.float32(thr))    # the list is the brute filter of the GPU's own planes ...
            want += hit.shape[0]
            for dm, i in hit:
                assert (int(dm), int(i) * D, int(g_w[dm, off + i])) in got
            near = np.abs(L["snr"] - thr) <= CMP.TIE    # ... and of the oracle's, outside 1e-3 of the threshold
            assert np.array_equal((gs >= np.float32(thr)) & ~near, (L["snr"] >= thr) & ~near)
        assert total == want
    return lv, infos


@pytest.mark.parametrize("n_dm,n_t,w0,levels", [(2, 4096, 16, 1), (2, 4096, 16, 4), (3, 5003, 16, 4), (1, 2049, 32, 3),
                                                (2, 1000, 16, 6), (1, 40, 16, 2), (2, 9001, 32, 8)])
def test_decimated_integer_data(P, n_dm, n_t, w0, levels):
    x = rng(500 + n_t).integers(-4, 6, size=(n_dm, n_t)).astype(np.float32)
    _run(P, x, w0, levels, "sqrt", O.Stats(0, 0.0, 0.0, 0.0, 1.0), thr=4.0)


@pytest.mark.parametrize("mode", ["sqrt", "linear", "anchored"])
@pytest.mark.parametrize("mu,sigma", [(0.0, 1.0), (100.0, 20.0)])
def test_decimated_noise_all_modes(P, mode, mu, sigma):
    x = (mu + sigma * rng(600).standard_normal((3, 7001))).astype(np.float32)
    x[1, 2000:2090] += 0.8 * sigma
    lv, infos = _run(P, x, 16, 4, mode, thr=5.0, stride=7008 if mode == "linear" else None)
    assert all(i["near_tie_rate"] < 0.08 for i in infos)


def test_decimated_on_grid_pulse_recovers_A_sqrt_W(P):
    n_t, A = 8192, 2.0
    for lvl, wp in [(1, 12), (2, 16), (3, 9)]:
        D, W, p = 1 << lvl, wp << lvl, 3200
        x = np.zeros((1, n_t), dtype=np.float32)
        x[0, p:p + W] = A
        lv, _ = _run(P, x, 16, 4, "sqrt", O.Stats(0, 0.0, 0.0, 0.0, 1.0))
        d = torch.from_numpy(x).cuda()
        snr, width = P.spd_boxcar_snr_decimated(d, P.write_stats(0.0, 1.0), 16, 4)
        off = P.decimated_level_offset(n_t, lvl)
        assert int(width[0, off + p // D].item()) == W
        assert float(snr[0, off + p // D].item()) == pytest.approx(A * math.sqrt(W), rel=3e-7)
        assert float(snr[torch.isfinite(snr)].max().item()) == pytest.approx(A * math.sqrt(W), rel=3e-7)


def test_decimated_level0_equals_the_exhaustive_sweep(P):
    x = rng(601).standard_normal((4, 6000)).astype(np.float32)
    d = torch.from_numpy(x).cuda()
    st = P.spd_stats(d)
    a, aw = P.spd_boxcar_snr(d, st, 16, "sqrt")
    b, bw = P.spd_boxcar_snr_decimated(d, st, 16, 3)
    assert torch.equal(a, b[:, :6000]) and torch.equal(aw.view(torch.int16), bw[:, :6000].view(torch.int16))


def test_decimated_config3_rows(P):
    """The SKA-like shape at Nmax = 128 as w0 = 16 x 4 levels on a row block of config 3, end to end with measured statistics;
    every injected pulse of those rows is still found (sensitivity >= sqrt(0.9) of the exhaustive search)."""
    cfg = gen.get_config(3)
    rows = sorted(set(gen.pulse_rows(cfg)[:12]) | set(range(0, 24)))
    x = gen.make_rows(cfg, rows)
    d = torch.from_numpy(x).cuda()
    st = P.spd_stats(d)
    g = P.read_stats(st)[0]
    o = O.stats(x)
    assert CMP.compare_stats(float(g["mean"]), float(g["sigma"]), o)
    lv, infos = _run(P, x, 16, 4, "sqrt", o, thr=cfg.threshold)
    exact_snr, _, _ = O.sweep(x, o.mean, O.sigma_table(o.sigma, float("nan"), 128, "sqrt"), want_margin=False)
    best_dec = np.max(np.stack([np.max(np.where(np.isfinite(L["snr"]), L["snr"], -np.inf), axis=1) for L in lv]), axis=0)
    best_exact = exact_snr.max(axis=1)
    strong = best_exact > 8.0
    assert strong.any() and np.all(best_dec[strong] >= 0.94 * best_exact[strong])


def test_decimated_argument_errors(P):
    x = torch.zeros((2, 4096), device="cuda")
    st = P.write_stats(0.0, 1.0)
    for w0, levels in [(8, 2), (16, 0), (16, 9), (32, 8 + 1), (24, 2)]:
        with pytest.raises(P.SpdError):
            P.spd_boxcar_snr_decimated(x, st, w0, levels)


# ---------------------------------------------------------------------------- fused decimated search (no planes)
def _run_fused(P, x, w0, levels, mode="sqrt", stats=None, thr=5.0, stride=None):
    """spd_search_fused_decimated against the candidate list of oracle O5 + O4 (level by level: set of (dm, t) outside 1e-3
    of the threshold, SNR tolerance, width / near-tie rules), and against the plane path's list (same (dm, t, snr) bits)."""
    from gpu_util import to_dev
    nmax = w0 << (levels - 1)
    o = O.full_stats(x, nmax if mode != "sqrt" else 0) if stats is None else stats
    st = P.write_stats(o.mean, o.sigma, o.sigma_nmax, o.nmax_of_sigma)
    d = to_dev(x, stride)
    out, cnt = P.spd_search_fused_decimated(d, st, w0, levels, mode, thr, capacity=1 << 20)
    rec, total = P.read_candidates(out, cnt)
    lv = O.sweep_decimated(x, o.mean, o.sigma, o.sigma_nmax, mode, w0, levels)
    sig_all = O.sigma_table(o.sigma, o.sigma_nmax, nmax, mode)
    r = CMP.compare_candidates_decimated(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 1 << 20, lv, w0, thr, x, o.mean, sig_all)
    assert r, str(r)
    snr, width = P.spd_boxcar_snr_decimated(d, st, w0, levels, mode)
    out2, cnt2 = P.spd_candidates_decimated(snr, width, x.shape[1], levels, thr, capacity=1 << 20)
    rec2, total2 = P.read_candidates(out2, cnt2)
    assert total == total2
    lvl = CMP.level_of_width(rec["width"], w0, levels)
    lvl2 = CMP.level_of_width(rec2["width"], w0, levels)
    a = np.lexsort((rec["t"], rec["dm"], lvl)); b = np.lexsort((rec2["t"], rec2["dm"], lvl2))
    for k in ("dm", "t", "snr"):
        assert rec[k][a].tobytes() == rec2[k][b].tobytes(), k
    assert (rec["width"][a] != rec2["width"][b]).mean() <= 0.02
    return rec, r.info


@pytest.mark.parametrize("n_dm,n_t,w0,levels", [(2, 4096, 16, 1), (2, 4096, 16, 4), (3, 5003, 16, 4), (1, 2049, 32, 3),
                                                (2, 1000, 16, 6), (1, 40, 16, 2), (2, 9001, 32, 8)])
def test_fused_decimated_integer_data(P, n_dm, n_t, w0, levels):
    x = rng(700 + n_t).integers(-4, 6, size=(n_dm, n_t)).astype(np.float32)
    rec, info = _run_fused(P, x, w0, levels, "sqrt", O.Stats(0, 0.0, 0.0, 0.0, 1.0), thr=4.0)
    assert info["gpu_hits"] > 0


@pytest.mark.parametrize("mode", ["sqrt", "linear", "anchored"])
@pytest.mark.parametrize("mu,sigma", [(0.0, 1.0), (100.0, 20.0)])
def test_fused_decimated_noise_all_modes(P, mode, mu, sigma):
    x = (mu + sigma * rng(800).standard_normal((3, 7001))).astype(np.float32)
    x[1, 2000:2090] += 0.8 * sigma
    rec, info = _run_fused(P, x, 16, 4, mode, thr=3.5, stride=7008 if mode == "linear" else None)
    assert info["gpu_hits"] > (30 if mode == "sqrt" else 3)       # eq. 5 flattens the SNR: fewer samples above the threshold


def test_fused_decimated_on_grid_pulse_and_overflow(P):
    n_t, A, W, p = 8192, 2.0, 48, 3200                      # 48 = 12 * 2^2
    x = np.zeros((1, n_t), dtype=np.float32); x[0, p:p + W] = A
    d = torch.from_numpy(x).cuda()
    out, cnt = P.spd_search_fused_decimated(d, P.write_stats(0.0, 1.0), 16, 4, "sqrt", 5.0, capacity=1 << 16)
    rec, total = P.read_candidates(out, cnt)
    k = int(np.argmax(rec["snr"]))
    assert (int(rec["t"][k]), int(rec["width"][k])) == (p, W) and float(rec["snr"][k]) == pytest.approx(A * math.sqrt(W), rel=3e-7)
    out, cnt = P.spd_search_fused_decimated(d, P.write_stats(0.0, 1.0), 16, 4, "sqrt", 5.0, capacity=8)   # overflow convention
    assert int(cnt.item()) == total > 8


def test_fused_decimated_linear_with_wrong_nmax_reports_misuse(P):
    x = torch.randn((2, 4096), device="cuda")
    st = P.spd_stats(x, 64)                                  # sigma_Nmax measured for 64, the search wants 128
    out, cnt = P.spd_search_fused_decimated(x, st, 16, 4, "linear", 5.0)
    with pytest.raises(P.SpdError):
        P.read_candidates(out, cnt)


def test_fused_decimated_config3_rows(P):
    cfg = gen.get_config(3)
    rows = sorted(set(gen.pulse_rows(cfg)[:12]) | set(range(0, 24)))
    x = gen.make_rows(cfg, rows)
    rec, info = _run_fused(P, x, 16, 4, "sqrt", O.stats(x), thr=cfg.threshold)
    assert info["gpu_hits"] > 0


@pytest.mark.parametrize("seed", range(4))
def test_random_decimated_cases_against_the_oracle(P, seed):
    """Seeded random shapes / w0 / levels / sigma modes / row strides through both decimated paths (planes + candidate pass,
    and the fused search); row lengths straddle the 1024-sample tiles (whole aligned tiles take the straight-line store path)."""
    r = np.random.default_rng(1611 + seed)
    done = 0
    while done < 8:
        n_dm = int(r.integers(1, 4))
        n_t = int(r.choice([r.integers(40, 1200), r.integers(1200, 9000), 4096, 8192, 3072 + 4 * int(r.integers(0, 300))]))
        w0 = int(r.choice([16, 32]))
        if n_t < w0:
            continue
        lmax = 1
        while lmax < 8 and (w0 << lmax) <= min(n_t, 4096):
            lmax += 1
        levels = int(r.integers(1, lmax + 1))
        mode = str(r.choice(["sqrt", "sqrt", "linear", "anchored"]))
        if n_dm * (n_t - (w0 << (levels - 1)) + 1) < 16:
            mode = "sqrt"
        mu, sg = float(r.choice([0.0, -50.0, 100.0])), float(r.choice([1.0, 0.1, 20.0]))
        x = (mu + sg * r.standard_normal((n_dm, n_t))).astype(np.float32)
        x[0, 20:20 + int(r.integers(1, min(30, n_t - 20)))] += 5 * sg
        stride = None if r.random() < 0.6 else n_t + int(r.integers(1, 9))
        thr = float(r.choice([3.0, 4.0, 5.0]))
        try:
            _run(P, x, w0, levels, mode, thr=thr, stride=stride)
            _run_fused(P, x, w0, levels, mode, thr=thr, stride=stride)
        except AssertionError as e:
            raise AssertionError(f"seed {seed} case {done}: {n_dm}x{n_t} w0 {w0} levels {levels} {mode} mu {mu} sigma {sg} stride {stride} thr {thr}: {e}")
        done += 1


def test_fused_decimated_search_is_cuda_graph_capturable(P):
    """spd_stats + spd_search_fused_decimated only enqueue work on the caller's stream and keep no state: captured once,
    replayed with the same result."""
    cfg = gen.get_config(1)
    x = torch.from_numpy(gen.make_array(cfg)).cuda()
    st, ws = P.new_stats("cuda"), P.new_workspace(cfg.n_dm, cfg.n_t, 32, "cuda")
    dws = torch.empty(int(P.lib().spd_decimated_workspace_bytes(cfg.n_dm, cfg.n_t, 16, 2)), dtype=torch.uint8, device="cuda")
    out, cnt = P.new_candidates(4096, "cuda")

    def step():
        P.spd_stats(x, 0, st, ws)
        P.spd_search_fused_decimated(x, st, 16, 2, "sqrt", cfg.threshold, out, cnt, ws=dws)

    step()
    torch.cuda.synchronize()
    n0 = int(cnt.item())
    ref = np.sort(out[:n0].cpu().numpy().view(P.CAND_DTYPE).reshape(-1), order=["dm", "t", "width"])
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        step()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            step()
    torch.cuda.synchronize()
    cnt.zero_(); out.zero_(); st.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert int(cnt.item()) == n0 > 0
    got = np.sort(out[:n0].cpu().numpy().view(P.CAND_DTYPE).reshape(-1), order=["dm", "t", "width"])
    assert got.tobytes() == ref.tobytes()


@pytest.mark.parametrize("mode", ["sqrt", "anchored"])
@pytest.mark.parametrize("mu,sigma", [(-1000.0, 1.0), (10000.0, 1.0), (3.0e5, 100.0)])
def test_decimated_baseline_far_above_the_noise(P, mode, mu, sigma):
    """|mu| = 1e3 .. 1e4 sigma through all 8 levels (Nmax 2048), planes and fused search: the level series are built from the
    mean-subtracted samples, so the SNR of the high levels must not pick up the rounding of D mu (ulp(256 * 1e4) = 0.25)."""
    x = (mu + sigma * rng(650).standard_normal((2, 20001))).astype(np.float32)
    x[1, 6000:7200] += np.float32(0.3 * sigma)              # a wide pulse for the top levels
    lv, infos = _run(P, x, 16, 8, mode, thr=5.0)
    assert lv[-1]["level"] == 7 and (lv[-1]["snr"] >= 5.0).any()
    rec, info = _run_fused(P, x, 16, 8, mode, thr=5.0)
    assert info["gpu_hits"] > 0 and (rec["width"] > 1024).any()
