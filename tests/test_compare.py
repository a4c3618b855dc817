"""-m "not gpu" tests of oracle/compare.py, the code that decides every parity verdict: it is fed the oracle's own
results with ONE injected error each and must reject every one of them, and must accept an fp32-rounded copy.
(SURVEY.md 8(c) "Comparator"; tolerances of BASELINE.json:north_star.)"""
import numpy as np
import pytest

from oracle import compare as CMP
from oracle import spd_oracle as O

NMAX, THR = 16, 2.5


@pytest.fixture(scope="module")
def case():
    rng = np.random.Generator(np.random.PCG64(77))
    x = rng.standard_normal((3, 4000)).astype(np.float32)
    x[1, 500:508] += 3.0
    x[2, 3990:3996] += 4.0                      # a pulse at the row end (truncated widths)
    x[0, 100:104] = 0.0                         # exact zeros: width ties of margin 0 at t = 100..103
    st = O.stats(x)
    sig = O.sigma_table(st.sigma, float("nan"), NMAX, "sqrt")
    snr, width, margin = O.sweep(x, st.mean, sig)
    dm, t, c_snr, c_w = O.candidates(snr, width, THR)
    return dict(x=x, mu=st.mean, sig=sig, snr=snr, width=width, margin=margin, dm=dm, t=t, c_snr=c_snr, c_w=c_w, st=st)


def _planes(c, g_snr=None, g_w=None):
    return CMP.compare_planes(c["x"], c["mu"], c["sig"], c["snr"].astype(np.float32) if g_snr is None else g_snr,
                              c["width"].astype(np.uint16) if g_w is None else g_w, c["snr"], c["width"], c["margin"])


def _cands(c, dm=None, t=None, s=None, w=None, count=None, capacity=1 << 16):
    dm = c["dm"] if dm is None else dm
    t = c["t"] if t is None else t
    s = c["c_snr"].astype(np.float32) if s is None else s
    w = c["c_w"] if w is None else w
    return CMP.compare_candidates(dm, t, s, w, len(dm) if count is None else count, capacity, c["snr"], c["width"],
                                  c["margin"], THR, c["x"], c["mu"], c["sig"])


def _near_tie(c):
    """A sample whose two best widths are closer than the tie tolerance, and the second-best width."""
    idx = np.argwhere((c["margin"] <= 0.5 * CMP.TIE) & (c["margin"] > 0))
    assert idx.size, "the fixture has no near-tie sample"
    for d, t in idx:
        wmax = min(NMAX, c["x"].shape[1] - t)
        s = O.snr_at(c["x"], c["mu"], c["sig"], [d] * wmax, [t] * wmax, np.arange(1, wmax + 1))
        order = np.argsort(-s)
        if order[0] + 1 == c["width"][d, t]:
            far = [k for k in range(wmax) if s[order[0]] - s[k] > 0.1]
            if far:
                return int(d), int(t), int(order[1] + 1), int(far[0] + 1)
    raise AssertionError("no usable near-tie sample")


# ------------------------------------------------------------------------------------------------- accepted
def test_fp32_rounded_copy_passes(case):
    assert _planes(case)
    assert len(case["dm"]) > 20
    r = _cands(case)
    assert r, str(r)


def test_any_candidate_order_passes(case):
    p = np.random.Generator(np.random.PCG64(5)).permutation(len(case["dm"]))
    r = _cands(case, case["dm"][p], case["t"][p], case["c_snr"][p].astype(np.float32), case["c_w"][p])
    assert r, str(r)


def test_second_best_width_inside_a_near_tie_passes(case):
    d, t, w2, _ = _near_tie(case)
    g_w = case["width"].astype(np.uint16).copy()
    g_w[d, t] = w2
    r = _planes(case, g_w=g_w)
    assert r and r.info["width_near_tie_exempt"] == 1, str(r)


def test_stats_within_tolerance_pass_and_outside_fail(case):
    st = case["st"]
    assert CMP.compare_stats(st.mean + 0.5e-6 * st.sigma, st.sigma * (1 + 0.5e-6), st)
    assert not CMP.compare_stats(st.mean + 3e-6 * max(abs(st.mean), st.sigma), st.sigma, st)
    assert not CMP.compare_stats(st.mean, st.sigma * (1 + 3e-6), st)
    assert not CMP.compare_stats(st.mean, float("nan"), st)
    st2 = O.Stats(st.n, st.T, st.S, st.mean, st.sigma, sigma_nmax=5.0, nmax_of_sigma=NMAX)
    assert CMP.compare_stats(st.mean, st.sigma, st2, 5.0 * (1 + 0.5e-6))
    assert not CMP.compare_stats(st.mean, st.sigma, st2, 5.0 * (1 + 3e-6))


# ------------------------------------------------------------------------------------------------- rejected: planes
def test_snr_off_by_twice_the_tolerance_is_rejected(case):
    g = case["snr"].astype(np.float32).copy()
    g[1, 777] += 2e-3
    r = _planes(case, g_snr=g)
    assert not r and r.info["snr_violations"] == 1


def test_relative_tolerance_applies_to_large_snr(case):
    g = case["snr"].astype(np.float32).copy()
    d, t = np.unravel_index(np.argmax(case["snr"]), case["snr"].shape)
    assert case["snr"][d, t] > 5
    g[d, t] *= np.float32(1 + 3e-4)              # 3e-4 relative of an SNR > 5 is above max(1e-3, 1e-4 |snr|)
    assert not _planes(case, g_snr=g)


def test_non_finite_snr_is_rejected(case):
    g = case["snr"].astype(np.float32).copy()
    g[0, 0] = np.nan
    assert not _planes(case, g_snr=g)


def test_wrong_width_at_a_clear_margin_is_rejected(case):
    d, t = np.argwhere(case["margin"] > 0.1)[0]
    g_w = case["width"].astype(np.uint16).copy()
    g_w[d, t] = g_w[d, t] % NMAX + 1
    assert not _planes(case, g_w=g_w)


def test_arbitrary_width_inside_a_near_tie_is_rejected(case):
    d, t, _, wfar = _near_tie(case)
    g_w = case["width"].astype(np.uint16).copy()
    g_w[d, t] = wfar                             # the margin is tiny, but THIS width is 0.1 below the best
    assert not _planes(case, g_w=g_w)


def test_width_that_does_not_fit_the_row_is_rejected(case):
    n_t = case["x"].shape[1]
    g_w = case["width"].astype(np.uint16).copy()
    t = n_t - 3
    g_w[0, t] = 9                                # only widths 1..3 fit; margin may or may not be a near-tie
    assert not _planes(case, g_w=g_w)


def test_shape_mismatch_is_rejected(case):
    assert not _planes(case, g_snr=case["snr"].astype(np.float32)[:, :-1])


# ------------------------------------------------------------------------------------------------- rejected: candidates
def _clear(c):
    """Index of a record that is neither near the threshold nor a width near-tie."""
    k = np.flatnonzero((np.abs(c["c_snr"] - THR) > 0.1) & (c["margin"][c["dm"], c["t"]] > 0.1))
    assert k.size
    return int(k[0])


def test_missing_candidate_is_rejected(case):
    k = _clear(case)
    keep = np.arange(len(case["dm"])) != k
    assert not _cands(case, case["dm"][keep], case["t"][keep], case["c_snr"][keep].astype(np.float32), case["c_w"][keep])


def test_extra_candidate_is_rejected(case):
    d, t = np.argwhere(case["snr"] < THR - 0.5)[0]
    assert not _cands(case, np.append(case["dm"], d), np.append(case["t"], t),
                      np.append(case["c_snr"], case["snr"][d, t]).astype(np.float32), np.append(case["c_w"], case["width"][d, t]))


def test_duplicate_candidate_is_rejected(case):
    k = _clear(case)
    assert not _cands(case, np.append(case["dm"], case["dm"][k]), np.append(case["t"], case["t"][k]),
                      np.append(case["c_snr"], case["c_snr"][k]).astype(np.float32), np.append(case["c_w"], case["c_w"][k]))


def test_out_of_range_candidate_is_rejected(case):
    dm = case["dm"].copy(); dm[0] = 3
    assert not _cands(case, dm=dm)
    t = case["t"].copy(); t[0] = case["x"].shape[1]
    assert not _cands(case, t=t)


def test_count_not_equal_to_list_length_is_rejected(case):
    assert not _cands(case, count=len(case["dm"]) + 1)


def test_overflow_is_rejected(case):
    assert not _cands(case, capacity=len(case["dm"]) - 1)


def test_candidate_snr_out_of_tolerance_is_rejected(case):
    k = _clear(case)
    s = case["c_snr"].astype(np.float32).copy()
    s[k] += 2e-3
    assert not _cands(case, s=s)


def test_candidate_wrong_width_at_a_clear_margin_is_rejected(case):
    k = _clear(case)
    w = case["c_w"].copy()
    w[k] = w[k] % NMAX + 1
    assert not _cands(case, w=w)


def test_candidate_arbitrary_width_inside_a_near_tie_is_rejected(case):
    """The hole VERDICT r1 named: inside a near-tie compare_candidates used to accept ANY width."""
    c = dict(case)
    d, t, w2, wfar = _near_tie(case)
    thr = float(case["snr"][d, t]) - 0.5         # make that sample a candidate
    dm, tt, cs, cw = O.candidates(case["snr"], case["width"], thr)
    k = int(np.flatnonzero((dm == d) & (tt == t))[0])

    def run(w):
        return CMP.compare_candidates(dm, tt, cs.astype(np.float32), w, len(dm), 1 << 20, case["snr"], case["width"],
                                      case["margin"], thr, case["x"], case["mu"], case["sig"])
    ok = cw.copy(); ok[k] = w2
    r = run(ok)
    assert r and r.info["width_near_tie_exempt"] == 1, str(r)
    bad = cw.copy(); bad[k] = wfar
    assert not run(bad)
    bad = cw.copy(); bad[k] = NMAX + 7           # a width that does not exist
    assert not run(bad)


def test_near_threshold_samples_are_exempt_either_way(case):
    d, t = np.unravel_index(np.argmin(np.abs(case["snr"] - 3.0)), case["snr"].shape)
    thr = float(case["snr"][d, t]) + 4e-4        # the oracle does not keep it, the fp32 side might
    dm, tt, cs, cw = O.candidates(case["snr"], case["width"], thr)
    args = (case["snr"], case["width"], case["margin"], thr, case["x"], case["mu"], case["sig"])
    assert CMP.compare_candidates(dm, tt, cs.astype(np.float32), cw, len(dm), 1 << 20, *args)
    r = CMP.compare_candidates(np.append(dm, d), np.append(tt, t), np.append(cs, case["snr"][d, t]).astype(np.float32),
                               np.append(cw, case["width"][d, t]), len(dm) + 1, 1 << 20, *args)
    assert r, str(r)


# ------------------------------------------------------------------------------------------------- decimated levels
@pytest.fixture(scope="module")
def dcase():
    rng = np.random.Generator(np.random.PCG64(78))
    x = rng.standard_normal((2, 3001)).astype(np.float32)
    x[1, 800:860] += 1.5
    st = O.stats(x)
    lv = O.sweep_decimated(x, st.mean, st.sigma, float("nan"), "sqrt", 16, 4)
    sig_all = O.sigma_table(st.sigma, float("nan"), 128, "sqrt")
    return dict(x=x, mu=st.mean, sig=sig_all, lv=lv)


def _lvl(c, l, g_snr=None, g_w=None):
    L = c["lv"][l]
    return CMP.compare_planes_level(c["x"], c["mu"], c["sig"], 16, L, L["snr"].astype(np.float32) if g_snr is None else g_snr,
                                    L["width"].astype(np.uint16) if g_w is None else g_w)


def test_level_planes_fp32_copy_passes(dcase):
    for l in range(4):
        r = _lvl(dcase, l)
        assert r, str(r)


def test_level_plane_errors_are_rejected(dcase):
    L = dcase["lv"][2]
    g = L["snr"].astype(np.float32).copy(); g[0, 10] += 2e-3
    assert not _lvl(dcase, 2, g_snr=g)
    w = L["width"].astype(np.uint16).copy()
    d, i = np.argwhere((L["margin"] > 0.1) & (L["width"] > 0))[0]
    w[d, i] = 36 if w[d, i] != 36 else 40
    assert not _lvl(dcase, 2, g_w=w)
    w = L["width"].astype(np.uint16).copy()
    w[0, L["snr"].shape[1] - 1] = 36                       # a position where no width of the level fits must stay (-inf, 0)
    assert not _lvl(dcase, 2, g_w=w)
    g = L["snr"].astype(np.float32).copy(); g[0, L["snr"].shape[1] - 1] = 0.0
    assert not _lvl(dcase, 2, g_snr=g)
    w = L["width"].astype(np.uint16).copy()
    cand = np.argwhere((L["margin"] <= CMP.TIE) & (L["width"] > 0))
    if cand.size:                                          # inside a near-tie: a width off the level's grid is still rejected
        d, i = cand[0]
        w[d, i] = 38
        assert not _lvl(dcase, 2, g_w=w)


# ------------------------------------------------------------------------------- candidate lists of the decimated search
def _dlist(c, thr=3.5):
    dm, t, sn, w, lv = O.candidates_decimated(c["lv"], thr)
    return dm, t, sn.astype(np.float32), w, lv


def _dcmp(c, dm, t, sn, w, thr=3.5, count=None, cap=1 << 20):
    return CMP.compare_candidates_decimated(dm, t, sn, w, len(dm) if count is None else count, cap, c["lv"], 16, thr,
                                            c["x"], c["mu"], c["sig"])


def test_level_of_width_partitions_the_grid():
    N = np.arange(0, 140)
    lv = CMP.level_of_width(N, 16, 4)
    assert np.array_equal(np.flatnonzero(lv == 0), np.arange(1, 17))
    assert np.array_equal(np.flatnonzero(lv == 1), np.arange(18, 33, 2))
    assert np.array_equal(np.flatnonzero(lv == 2), np.arange(36, 65, 4))
    assert np.array_equal(np.flatnonzero(lv == 3), np.arange(72, 129, 8))
    assert lv[0] == -1 and lv[17] == -1 and lv[34] == -1 and lv[130] == -1


def test_decimated_list_fp32_copy_passes_in_any_order(dcase):
    dm, t, sn, w, lv = _dlist(dcase)
    assert dm.size > 50 and len(set(lv.tolist())) == 4      # every level contributes
    r = _dcmp(dcase, dm, t, sn, w)
    assert r, str(r)
    p = np.random.Generator(np.random.PCG64(5)).permutation(dm.size)
    assert _dcmp(dcase, dm[p], t[p], sn[p], w[p])


def test_decimated_list_errors_are_rejected(dcase):
    dm, t, sn, w, lv = _dlist(dcase)
    L2 = dcase["lv"][2]
    k = int(np.flatnonzero((lv == 2) & (np.abs(sn - 3.5) > 0.05))[0])
    for name, mut in [
        ("missing", lambda a: tuple(np.delete(v, k) for v in a)),
        ("duplicate", lambda a: tuple(np.append(v, v[k]) for v in a)),
        ("snr", lambda a: (a[0], a[1], np.where(np.arange(a[2].size) == k, a[2] + 2e-3, a[2]).astype(np.float32), a[3])),
        ("t not on the level's grid", lambda a: (a[0], np.where(np.arange(a[1].size) == k, a[1] + 1, a[1]), a[2], a[3])),
        ("width off every grid", lambda a: (a[0], a[1], a[2], np.where(np.arange(a[3].size) == k, 34, a[3]))),
    ]:
        m = mut((dm, t, sn, w))
        assert not _dcmp(dcase, *m), name
    # a record moved to another level's grid by its width is an extra there and a miss here
    w2 = w.copy(); w2[k] = 20
    assert not _dcmp(dcase, dm, t, sn, w2)
    # wrong width of the same level at a clear margin
    i = t // 4
    clear = np.flatnonzero((lv == 2) & (L2["margin"][dm, np.minimum(i, L2["snr"].shape[1] - 1)] > 0.1))
    assert clear.size
    w3 = w.copy(); w3[clear[0]] = 36 if w[clear[0]] != 36 else 40
    assert not _dcmp(dcase, dm, t, sn, w3)
    assert not _dcmp(dcase, dm, t, sn, w, count=dm.size + 1)
    assert not _dcmp(dcase, dm, t, sn, w, cap=dm.size - 1)
    # an extra record below the threshold
    d, ii = np.argwhere((L2["snr"] < 3.0) & (L2["width"] > 0))[0]
    assert not _dcmp(dcase, np.append(dm, d), np.append(t, ii * 4), np.append(sn, np.float32(L2["snr"][d, ii])), np.append(w, L2["width"][d, ii]))
