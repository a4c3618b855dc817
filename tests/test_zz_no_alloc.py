"""spd_stats_rows_noalloc: the per-row statistics for callers that cannot allocate device memory.

The callers in question are detection stages embedded in a real-time pipeline that owns the whole card: the framework
gives a stage the device buffers it reads and writes and forbids cudaMalloc (all memory is already in the framework's
pools, and an allocation would make the device wait and stall the other stages).  The entry point therefore keeps its
block partials in a 3 MiB static device array inside libspd.so and takes only the caller's input and output.

What is checked here: its output against the existing path (spd_stats_rows with a caller workspace) on TWO calls in a row.
The second call has fewer rows, another length and another sigma_Nmax request, so anything it wrongly picked up from
what the first call left in the shared array would show.  Tolerance: the statistics tolerance of the parity tests
(oracle.compare.STAT_REL = 1e-6 relative); the two paths run the same kernels, so the bytes are compared as well.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests),
and it passes on its own in a fresh process as well as after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle.compare import STAT_REL


@pytest.fixture(scope="module")
def P():
    import paper_1611_09704_b200 as P
    from paper_1611_09704_b200 import build as B
    B.ensure_built()
    P.lib()
    return P


def _rows(seed, n_dm, n_t):
    """Rows with their own baseline and noise level each (the data per-row statistics exist for)."""
    r = np.random.Generator(np.random.PCG64(seed))
    mu = r.uniform(-50, 50, n_dm)
    sg = 10.0 ** r.uniform(-1, 1, n_dm)
    return (mu[:, None] + sg[:, None] * r.standard_normal((n_dm, n_t))).astype(np.float32)


def _close(a, b, what):
    assert np.all(np.abs(a - b) <= STAT_REL * np.maximum(np.abs(b), 1e-300)), f"{what}: {a} vs {b}"


@pytest.mark.gpu
def test_noalloc_matches_the_workspace_path_on_two_calls_in_a_row(P):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    cases = [(_rows(1, 96, 20000), 0), (_rows(2, 7, 9001), 64)]          # (x, nmax_for_sigma): call 1, then call 2
    dev = [torch.from_numpy(x).cuda() for x, _ in cases]
    # everything the caller owns exists before the first call: the entry point gets inputs and outputs only
    outs = [torch.zeros(x.shape[0] * P.STATS_DTYPE.itemsize, dtype=torch.uint8, device="cuda") for x, _ in cases]
    got = []
    for d, o, (_, nsig) in zip(dev, outs, cases):                        # two calls back to back on one stream
        P.spd_stats_rows_noalloc(d, o, nsig)
    for o in outs:
        got.append(P.read_stats(o))
    for d, g, (x, nsig) in zip(dev, got, cases):
        want = P.read_stats(P.spd_stats_rows(d, nsig))                   # the existing path, its own workspace
        assert np.array_equal(g["n"], want["n"]) and np.all(g["n"] == x.shape[1])
        assert np.array_equal(g["nmax_of_sigma"], want["nmax_of_sigma"]) and np.all(g["nmax_of_sigma"] == nsig)
        tol_mu = STAT_REL * np.maximum(np.abs(want["mean"]), want["sigma"])
        assert np.all(np.abs(g["mean"] - want["mean"]) <= tol_mu)
        _close(g["sigma"], want["sigma"], "sigma")
        if nsig:
            _close(g["sigma_nmax"], want["sigma_nmax"], "sigma_nmax")
        assert g.tobytes() == want.tobytes()                             # same kernels, same order of merges
        # and the numbers mean something: each row's mean and sigma against numpy in float64
        _close(g["sigma"], x.astype(np.float64).std(axis=1), "sigma vs numpy")


@pytest.mark.gpu
def test_noalloc_refuses_more_rows_than_its_scratch_holds(P):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    n_dm = P.noalloc_max_rows() + 1
    x = torch.zeros((n_dm, 64), dtype=torch.float32, device="cuda")
    out = torch.full((n_dm * P.STATS_DTYPE.itemsize,), 0xAB, dtype=torch.uint8, device="cuda")
    with pytest.raises(P.SpdError, match="NOALLOC_LIMIT"):
        P.spd_stats_rows_noalloc(x, out)
    torch.cuda.synchronize()
    assert bool((out == 0xAB).all())                                     # nothing was launched
    ok = P.read_stats(P.spd_stats_rows_noalloc(x[:P.noalloc_max_rows()], out[:P.noalloc_max_rows() * 80]))
    assert np.all(ok["n"] == 64) and np.all(ok["mean"] == 0.0)           # exactly the maximum is accepted


def test_noalloc_limit_is_checked_before_the_device_is_touched(P):
    """No GPU needed: the row limit and the argument checks come before any CUDA call."""
    L = P.lib()
    assert L.spd_stats_rows_noalloc_max_rows() == 8192
    fake = C.c_void_p(256)
    assert L.spd_stats_rows_noalloc(fake, 8193, 100, 100, 0, fake, None) == 4
    assert b"NOALLOC_LIMIT" in L.spd_status_string(4)
    assert L.spd_stats_rows_noalloc(None, 4, 100, 100, 0, fake, None) == 1
    assert L.spd_stats_rows_noalloc(fake, 4, 100, 100, 0, None, None) == 1
    assert L.spd_stats_rows_noalloc(fake, 4, 100, 99, 0, fake, None) == 1
    assert L.spd_stats_rows_noalloc(fake, 4, 100, 100, 101, fake, None) == 1
