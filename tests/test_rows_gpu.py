"""-m gpu parity of the per-DM-row statistics path (spd_stats_rows, spd_boxcar_snr_rows, spd_search_fused_rows;
PAPER.md:44, reading A3's alternative) against oracle O3r, element by element."""
import numpy as np
import pytest
import torch

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


def hetero(seed, n_dm, n_t):
    """Rows with very different baselines and noise levels: one global (mu, sigma) would be useless here."""
    r = np.random.Generator(np.random.PCG64(seed))
    mu = r.uniform(-200, 200, n_dm)
    sg = 10.0 ** r.uniform(-1, 1.5, n_dm)
    x = (mu[:, None] + sg[:, None] * r.standard_normal((n_dm, n_t))).astype(np.float32)
    for d in range(0, n_dm, 2):
        p = int(r.integers(0, max(1, n_t - 40)))
        x[d, p:p + 24] += 2.0 * sg[d]
    return x


@pytest.mark.parametrize("n_dm,n_t,nsig,stride", [(5, 3000, 0, None), (7, 20000, 16, None), (3, 4097, 64, 4100), (70, 700, 0, None),
                                                  (2, 40000, 512, None)])
def test_stats_rows_parity(P, n_dm, n_t, nsig, stride):
    from gpu_util import to_dev
    x = hetero(10 + n_dm, n_dm, n_t)
    g = P.read_stats(P.spd_stats_rows(to_dev(x, stride), nsig))
    o = O.stats_rows(x, nsig)
    for d in range(n_dm):
        assert int(g["n"][d]) == n_t and int(g["nmax_of_sigma"][d]) == nsig
        r = CMP.compare_stats(float(g["mean"][d]), float(g["sigma"][d]), o[d], float(g["sigma_nmax"][d]) if nsig else None)
        assert r, f"row {d}: {r}"


@pytest.mark.parametrize("nmax,mode", [(8, "sqrt"), (32, "sqrt"), (128, "sqrt"), (100, "sqrt"), (24, "linear"), (64, "anchored"), (300, "linear")])
def test_sweep_and_fused_search_with_row_statistics(P, nmax, mode):
    from gpu_util import to_dev
    n_dm, n_t = 6, 5000
    x = hetero(20 + nmax, n_dm, n_t)
    nsig = nmax if mode != "sqrt" else 0
    o = O.stats_rows(x, nsig)
    a = np.zeros(n_dm, dtype=P.STATS_DTYPE)                  # the same statistics on both sides: isolates the sweep
    for d in range(n_dm):
        a["mean"][d], a["sigma"][d], a["sigma_nmax"][d], a["nmax_of_sigma"][d] = o[d].mean, o[d].sigma, o[d].sigma_nmax, nsig
    st = torch.from_numpy(a.view(np.uint8).copy()).cuda()
    d_x = to_dev(x)
    snr, width = P.spd_boxcar_snr_rows(d_x, st, nmax, mode)
    o_snr, o_w, o_m, sig = O.sweep_rows(x, o, nmax, mode)
    g_snr, g_w = snr.cpu().numpy(), width.cpu().numpy()
    thr = 5.0 if mode == "sqrt" else 3.5                 # eq. 5 as printed roughly halves the SNR of the wide widths
    out, cnt = P.spd_search_fused_rows(d_x, st, nmax, mode, thr, capacity=1 << 16)
    rec, total = P.read_candidates(out, cnt)
    assert total > 0
    for d in range(n_dm):                                    # row by row: each has its own mu and sigma_w table
        r = CMP.compare_planes(x[d:d + 1], o[d].mean, sig[d], g_snr[d:d + 1], g_w[d:d + 1], o_snr[d:d + 1], o_w[d:d + 1], o_m[d:d + 1])
        assert r, f"row {d}: {r}"
        m = rec["dm"] == d
        rc = CMP.compare_candidates(np.zeros(int(m.sum()), dtype=np.int64), rec["t"][m], rec["snr"][m], rec["width"][m], int(m.sum()), 1 << 16,
                                    o_snr[d:d + 1], o_w[d:d + 1], o_m[d:d + 1], thr, x[d:d + 1], o[d].mean, sig[d])
        assert rc, f"row {d}: {rc}"


def test_row_statistics_end_to_end_find_pulses_a_global_estimate_misses(P):
    """stats_rows -> sweep_rows -> candidates on the GPU: with per-row statistics the 2-sigma-per-sample pulse of a quiet row
    is found although the array's global sigma (dominated by the loud rows) would bury it."""
    n_dm, n_t = 8, 30000
    x = hetero(33, n_dm, n_t)
    d_x = torch.from_numpy(x).cuda()
    st = P.spd_stats_rows(d_x)
    snr, width = P.spd_boxcar_snr_rows(d_x, st, 32, "sqrt")
    out, cnt = P.spd_candidates(snr, width, 7.0, capacity=1 << 16)
    rec, total = P.read_candidates(out, cnt)
    assert set(range(0, n_dm, 2)) <= set(rec["dm"].tolist())      # every pulse-bearing row reports
    g = P.read_stats(P.spd_stats(d_x))[0]
    quiet = int(np.argmin(P.read_stats(st)["sigma"][::2])) * 2
    snr_g, _ = P.spd_boxcar_snr(d_x, P.spd_stats(d_x), 32, "sqrt")
    assert float(snr_g[quiet].max()) < 7.0 or float(g["sigma"]) < 2 * float(P.read_stats(st)["sigma"][quiet])
