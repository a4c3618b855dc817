"""Seeded random shapes / widths / sigma modes / row strides through spd_stats, spd_boxcar_snr, spd_candidates and
spd_search_fused, each compared with the oracle under the tolerances of DESIGN.md section 5.  The width list straddles
every kernel switch (narrow kernel up to 24, 64-thread CTAs up to 256, blocks of 8 widths) and the row lengths every
tile edge (1024- and 2048-sample tiles)."""
import numpy as np
import pytest
import torch

from oracle import compare as CMP
from oracle import spd_oracle as O

pytestmark = pytest.mark.gpu

WIDTHS = [1, 2, 7, 8, 9, 16, 23, 24, 25, 31, 32, 33, 64, 100, 128, 129, 255, 256, 257, 300, 512, 700]


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1611_09704_b200 as P
    from paper_1611_09704_b200 import build as B
    B.ensure_built()
    P.lib()
    return P


@pytest.mark.parametrize("seed", range(8))
def test_random_cases_against_the_oracle(P, seed):
    from gpu_util import gpu_candidates, gpu_fused, to_dev
    rng = np.random.default_rng(9704 + seed)
    done = 0
    while done < 12:
        n_dm = int(rng.integers(1, 5))
        n_t = int(rng.choice([rng.integers(8, 40), rng.integers(40, 3000), rng.integers(3000, 12000)]))
        nmax = int(min(n_t, rng.choice(WIDTHS)))
        mode = str(rng.choice(["sqrt", "sqrt", "linear", "anchored"]))
        if n_dm * (n_t - nmax + 1) < 16:
            mode = "sqrt"                                # sigma_Nmax of a handful of windows is degenerate
        mu, sg = float(rng.choice([0.0, 3.0, -50.0, 100.0])), float(rng.choice([1.0, 0.1, 20.0]))
        x = (mu + sg * rng.standard_normal((n_dm, n_t))).astype(np.float32)
        if n_t > 50:
            x[0, 20:20 + int(rng.integers(1, 30))] += 6 * sg
        stride = None if rng.random() < 0.6 else n_t + int(rng.integers(1, 9))
        thr = float(rng.choice([2.0, 4.0, 6.0]))
        tag = f"seed {seed} case {done}: {n_dm}x{n_t} nmax {nmax} {mode} mu {mu} sigma {sg} stride {stride} thr {thr}"
        nsig = nmax if mode != "sqrt" else 0
        o = O.full_stats(x, nsig)
        d = to_dev(x, stride)
        g = P.read_stats(P.spd_stats(d, nsig))[0]
        r = CMP.compare_stats(float(g["mean"]), float(g["sigma"]), o, float(g["sigma_nmax"]) if nsig else None)
        assert r, tag + " " + str(r)
        sig = O.sigma_table(o.sigma, o.sigma_nmax, nmax, mode)
        st = P.write_stats(o.mean, o.sigma, o.sigma_nmax if nsig else float("nan"), nsig)     # same statistics on both sides
        snr, width = P.spd_boxcar_snr(d, st, nmax, mode)
        o_snr, o_w, o_m = O.sweep(x, o.mean, sig)
        r = CMP.compare_planes(x, o.mean, sig, snr.cpu().numpy(), width.cpu().numpy(), o_snr, o_w, o_m)
        assert r, tag + " " + str(r)
        rec, total = gpu_candidates(snr, width, thr, capacity=1 << 18)
        r = CMP.compare_candidates(rec["dm"], rec["t"], rec["snr"], rec["width"], total, 1 << 18, o_snr, o_w, o_m, thr, x, o.mean, sig)
        assert r, tag + " " + str(r)
        rec2, total2 = gpu_fused(d, st, nmax, mode, thr, capacity=1 << 18)
        r = CMP.compare_candidates(rec2["dm"], rec2["t"], rec2["snr"], rec2["width"], total2, 1 << 18, o_snr, o_w, o_m, thr, x, o.mean, sig)
        assert r and total2 == total, tag + " " + str(r)
        done += 1
