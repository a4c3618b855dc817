"""-m "not gpu" pins of oracle O5 (decimation in time + boxcar, reading A20 of DESIGN.md).

None of them re-types the oracle's loop: level 0 must reduce to the pinned exhaustive oracle O3, the decimated series
to a plain block sum, every level to an explicit O(n W0 D) inner sum over the ORIGINAL samples, an on-grid rectangular
pulse to its closed form A sqrt(W), and an off-grid one must stay within the sensitivity bound the width grid implies."""
import math

import numpy as np
import pytest

from oracle import spd_oracle as O

W0, LEVELS = 16, 4                    # Nmax = 128: 1..16 | 18..32 step 2 | 36..64 step 4 | 72..128 step 8
NMAX = W0 << (LEVELS - 1)


def rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def test_width_grid():
    g = O.decimated_levels(W0, LEVELS)
    assert g == [(0, 1, 1, 16), (1, 2, 9, 16), (2, 4, 9, 16), (3, 8, 9, 16)]
    widths = sorted(w * D for (_, D, lo, hi) in g for w in range(lo, hi + 1))
    assert widths == list(range(1, 17)) + list(range(18, 33, 2)) + list(range(36, 65, 4)) + list(range(72, 129, 8))
    assert len(set(widths)) == len(widths)          # no effective width is searched twice


def test_level0_is_the_exhaustive_oracle():
    x = (3.0 + 2.0 * rng(1).standard_normal((3, 777))).astype(np.float32)
    st = O.stats(x)
    lv = O.sweep_decimated(x, st.mean, st.sigma, float("nan"), "sqrt", W0, LEVELS)
    snr, width, margin = O.sweep(x, st.mean, O.sigma_table(st.sigma, float("nan"), W0, "sqrt"))
    assert np.array_equal(lv[0]["snr"], snr) and np.array_equal(lv[0]["width"], width)
    assert np.array_equal(lv[0]["margin"], margin)


def test_decimated_series_is_a_block_sum_and_floors_odd_lengths():
    x = rng(2).integers(-5, 6, size=(2, 1003)).astype(np.float32)
    lv = O.sweep_decimated(x, 0.0, 1.0, float("nan"), "sqrt", W0, LEVELS)
    n = 1003
    for l in lv:
        D = l["D"]
        n_l = n >> l["level"]                       # floor at every level == floor(n / 2^l)
        assert l["x"].shape == (2, n_l)
        want = x[:, :n_l * D].astype(np.float64).reshape(2, n_l, D).sum(axis=2)
        assert np.array_equal(l["x"], want)


@pytest.mark.parametrize("mode", ["sqrt", "linear", "anchored"])
def test_every_level_against_explicit_sums_over_the_original_samples(mode):
    n = 300
    x = rng(3).integers(-3, 5, size=(2, n)).astype(np.float32)
    mu, sigma, snm = 0.5, 1.5, 40.0
    sig = O.sigma_table(sigma, snm, NMAX, mode)
    lv = O.sweep_decimated(x, mu, sigma, snm, mode, W0, LEVELS)
    xd = x.astype(np.float64)
    for l in lv:
        D, lvl = l["D"], l["level"]
        n_l = n >> lvl
        wmin = 1 if lvl == 0 else W0 // 2 + 1
        for d in range(2):
            for i in range(n_l):
                best, W = -math.inf, 0
                for w in range(wmin, W0 + 1):
                    if i + w > n_l:
                        break
                    N = w * D
                    s = (xd[d, i * D:i * D + N].sum() - N * mu) / sig[N - 1]
                    if s > best:
                        best, W = s, N
                assert l["width"][d, i] == W, (lvl, d, i)
                if W == 0:
                    assert l["snr"][d, i] == -math.inf
                else:
                    assert l["snr"][d, i] == pytest.approx(best, rel=1e-13, abs=1e-13)


def test_positions_where_no_width_of_the_level_fits():
    x = np.ones((1, 64), dtype=np.float32)
    lv = O.sweep_decimated(x, 0.0, 1.0, float("nan"), "sqrt", W0, 3)
    l1 = lv[1]                                      # n_1 = 32, widths 9..16: the last 8 positions see none
    assert np.all(l1["width"][0, :24] > 0) and np.all(l1["width"][0, 24:] == 0) and np.all(np.isinf(l1["snr"][0, 24:]))
    assert l1["width"][0, 23] == 18 and l1["width"][0, 16] == 32      # constant input: the widest width that fits wins
    l2 = lv[2]                                      # n_2 = 16, widths 9..16 decimated = 36..64
    assert l2["width"][0, 0] == 64 and l2["width"][0, 7] == 36 and l2["width"][0, 8] == 0


@pytest.mark.parametrize("lvl,wprime", [(0, 5), (1, 9), (1, 16), (2, 11), (3, 16), (3, 9)])
def test_on_grid_rectangular_pulse_recovers_A_sqrt_W(lvl, wprime):
    """Figure-1 property on the decimated grid: a pulse of width W = w' 2^l starting on the level's time grid is matched
    exactly by one boxcar of that level, SNR = A sqrt(W), and nothing on any level exceeds it."""
    D = 1 << lvl
    W, A, n = wprime * D, 2.0, 2048
    p = 40 * 8                                      # on the grid of every level
    x = np.zeros((1, n), dtype=np.float32)
    x[0, p:p + W] = A
    lv = O.sweep_decimated(x, 0.0, 1.0, float("nan"), "sqrt", W0, LEVELS)
    l = lv[lvl]
    assert l["width"][0, p // D] == W
    assert l["snr"][0, p // D] == pytest.approx(A * math.sqrt(W), rel=1e-14)
    top = max(float(np.max(q["snr"])) for q in lv)
    assert top == pytest.approx(A * math.sqrt(W), rel=1e-14)


def sensitivity_table():
    """Worst-case (over the start offset) ratio of the best decimated SNR to the matched-filter SNR A sqrt(W) of a
    noiseless rectangular pulse, for every W = 1..Nmax."""
    A, n = 1.0, 1024
    worst = {}
    for W in range(1, NMAX + 1):
        ratios = []
        for off in range(8):                        # the coarsest time grid has period 8
            x = np.zeros((1, n), dtype=np.float32)
            p = 400 + off
            x[0, p:p + W] = A
            lv = O.sweep_decimated(x, 0.0, 1.0, float("nan"), "sqrt", W0, LEVELS)
            ratios.append(max(float(np.max(q["snr"])) for q in lv) / (A * math.sqrt(W)))
        worst[W] = min(ratios)
        assert max(ratios) <= 1.0 + 1e-12           # a boxcar cannot beat the matched filter
    return worst


def test_off_grid_sensitivity_loss_is_bounded():
    """The price of the coarser grid (Keane & Petroff): tabulated in DESIGN.md section 2 (A20).
    Widths up to W0 lose nothing; above, the loss is bounded by the grid (step 2^l in width and in start time)."""
    worst = sensitivity_table()
    assert all(worst[W] == pytest.approx(1.0, abs=1e-12) for W in range(1, W0 + 1))
    assert min(worst.values()) > 0.90
    band = lambda lo, hi: min(worst[W] for W in range(lo, hi + 1))
    assert band(17, 32) > 0.94 and band(33, 64) > 0.92 and band(65, 128) > 0.90


def test_eq5_levels_use_sigma_of_the_effective_width():
    x = np.zeros((1, 256), dtype=np.float32)
    x[0, 64:64 + 48] = 1.0                           # W = 48 = 12 * 4: on the grid of level 2
    sigma, snm = 2.0, 30.0
    lv = O.sweep_decimated(x, 0.0, sigma, snm, "linear", W0, LEVELS)
    want = 48.0 / (math.sqrt(48) * sigma + 47 * snm / (NMAX - 1))       # eq. 5 at N = 48 with Nmax = 128
    assert lv[2]["snr"][0, 16] == pytest.approx(want, rel=1e-14) and lv[2]["width"][0, 16] == 48


def test_candidate_list_of_the_decimated_search():
    """O4 over the levels of O5: with one level it is the exhaustive search's list; in general it is the brute filter of
    every level plane with t = i 2^l; an on-grid rectangular pulse heads the list at (p, W) with SNR A sqrt(W)."""
    r = np.random.Generator(np.random.PCG64(91))
    x = r.standard_normal((3, 4100)).astype(np.float32)
    a = O.search_decimated(x, 16, 1, "sqrt", 3.0)
    b = O.search(x, 16, "sqrt", 3.0)
    for u, v in zip(a["cand"][:4], b["cand"]):
        assert np.array_equal(u, v)
    c = O.search_decimated(x, 16, 4, "sqrt", 3.0)
    dm, t, snr, w, lv = c["cand"]
    want = 0
    got = set(zip(dm.tolist(), t.tolist(), w.tolist()))
    assert len(got) == dm.size
    for L in c["levels"]:
        hit = np.argwhere(L["snr"] >= 3.0)
        want += hit.shape[0]
        for d, i in hit:
            assert (int(d), int(i) * L["D"], int(L["width"][d, i])) in got
    assert want == dm.size and np.all(snr >= 3.0)
    A, W, p = 2.0, 48, 1024                                   # 48 = 12 * 2^2: on the grid of level 2
    x = np.zeros((1, 4096), dtype=np.float32); x[0, p:p + W] = A
    lv = O.sweep_decimated(x, 0.0, 1.0, float("nan"), "sqrt", 16, 4)
    dm, t, snr, w, l = O.candidates_decimated(lv, 5.0)
    k = int(np.argmax(snr))
    assert (int(t[k]), int(w[k]), int(l[k])) == (p, W, 2) and snr[k] == pytest.approx(A * np.sqrt(W), rel=1e-12)
