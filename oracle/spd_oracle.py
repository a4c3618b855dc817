"""ctypes front end of oracle/spd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports paper_1611_09704_b200 and shares nothing with it.

Each wrapper cites the PAPER.md passage its C function follows; see the C file for the
formulae.  All arithmetic is float64 on the CPU.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spd_oracle.c")
_LIB = os.path.join(_HERE, "libspd_oracle.so")
_lib = None

MODE_SQRT, MODE_LINEAR, MODE_LINEAR_ANCHORED = 0, 1, 2
_MODES = {"sqrt": 0, "linear": 1, "anchored": 2, 0: 0, 1: 1, 2: 2}


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (plain -O2, OpenMP over rows only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        i64, dbl, i32 = C.c_int64, C.c_double, C.c_int
        P = C.c_void_p
        L.spd_oracle_stats.argtypes = [P, i64, i64, i64, i64, P]
        L.spd_oracle_merge.argtypes = [P, P]
        L.spd_oracle_chan_run.argtypes = [P, i64, P]
        L.spd_oracle_sigma_nmax.argtypes = [P, i64, i64, i64, i32, i64, P]
        L.spd_oracle_sigma_table.argtypes = [dbl, dbl, i32, i32, P]
        L.spd_oracle_sweep.argtypes = [P, i64, i64, i64, dbl, P, i32, P, P, P]
        L.spd_oracle_snr_fixed_width.argtypes = [P, i64, i64, i64, dbl, dbl, i32, P]
        L.spd_oracle_snr_at.argtypes = [P, i64, i64, dbl, P, i32, P, P, P, i64, P]
        L.spd_oracle_sweep_rows.argtypes = [P, i64, i64, i64, P, P, i32, P, P, P]
        L.spd_oracle_sweep_rows.restype = None
        L.spd_oracle_sweep_level.argtypes = [P, i64, i64, dbl, P, i32, i32, i32, P, P, P]
        L.spd_oracle_sweep_level.restype = None
        L.spd_oracle_decimate2.argtypes = [P, i64, i64, P]
        L.spd_oracle_decimate2.restype = None
        L.spd_oracle_candidates.argtypes = [P, P, i64, i64, dbl, i64, P, P, P, P]
        L.spd_oracle_candidates.restype = i64
        for f in ("spd_oracle_stats", "spd_oracle_merge", "spd_oracle_chan_run", "spd_oracle_sigma_nmax",
                  "spd_oracle_sigma_table", "spd_oracle_sweep", "spd_oracle_snr_fixed_width", "spd_oracle_snr_at"):
            getattr(L, f).restype = None
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _as_x(x: np.ndarray) -> Tuple[np.ndarray, int, int, int]:
    assert x.dtype == np.float32 and x.ndim == 2 and x.strides[1] == 4, "x must be float32 [n_dm][n_t], time fastest"
    assert x.strides[0] % 4 == 0
    return x, x.shape[0], x.shape[1], x.strides[0] // 4


@dataclass
class Stats:
    n: int
    T: float
    S: float
    mean: float
    sigma: float
    sigma_nmax: float = float("nan")
    nmax_of_sigma: int = 0


def stats(x: np.ndarray, block: int = 1000) -> Stats:
    """O1: eq. 1 per block of `block` samples, blocks folded left to right with eq. 2."""
    x, n_dm, n_t, rs = _as_x(x)
    out = np.zeros(5, dtype=np.float64)
    _load().spd_oracle_stats(_p(x), n_dm, n_t, rs, block, _p(out))
    return Stats(int(out[0]), float(out[1]), float(out[2]), float(out[3]), float(out[4]))


def chan_run(v: np.ndarray) -> np.ndarray:
    """eq. 1 over a float64 vector -> [m, T, S]."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.zeros(3, dtype=np.float64)
    _load().spd_oracle_chan_run(_p(v), v.size, _p(out))
    return out


def merge(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """eq. 2 as printed: [m,T,S] (+) [n,T,S]."""
    a = np.array(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    _load().spd_oracle_merge(_p(a), _p(b))
    return a


def sigma_nmax(x: np.ndarray, nmax: int, block: int = 1000) -> Stats:
    """O1b: population std of the Nmax-sample boxcar SUMS over all full windows."""
    x, n_dm, n_t, rs = _as_x(x)
    out = np.zeros(5, dtype=np.float64)
    _load().spd_oracle_sigma_nmax(_p(x), n_dm, n_t, rs, int(nmax), block, _p(out))
    return Stats(int(out[0]), float(out[1]), float(out[2]), float(out[3]), float(out[4]))


def full_stats(x: np.ndarray, nmax_for_sigma: int = 0) -> Stats:
    """stats() plus, when nmax_for_sigma > 0, the true sigma_Nmax needed by eq. 5."""
    s = stats(x)
    if nmax_for_sigma > 0:
        s.sigma_nmax = sigma_nmax(x, nmax_for_sigma).sigma
        s.nmax_of_sigma = int(nmax_for_sigma)
    return s


def sigma_table(sigma: float, sig_nmax: float, nmax: int, mode) -> np.ndarray:
    """O2: sigma_w for w = 1..nmax by eq. 4 / eq. 5 / anchored variant."""
    out = np.zeros(int(nmax), dtype=np.float64)
    _load().spd_oracle_sigma_table(float(sigma), float(sig_nmax), int(nmax), _MODES[mode], _p(out))
    return out


def sweep(x: np.ndarray, mu: float, sig: np.ndarray, want_margin: bool = True):
    """O3: Algorithm 1 as repaired: returns (snr f64, width i32, margin f64|None)."""
    x, n_dm, n_t, rs = _as_x(x)
    sig = np.ascontiguousarray(sig, dtype=np.float64)
    snr = np.empty((n_dm, n_t), dtype=np.float64)
    width = np.empty((n_dm, n_t), dtype=np.int32)
    margin = np.empty((n_dm, n_t), dtype=np.float64) if want_margin else None
    _load().spd_oracle_sweep(_p(x), n_dm, n_t, rs, float(mu), _p(sig), sig.size, _p(snr), _p(width), _p(margin))
    return snr, width, margin


def snr_fixed_width(x: np.ndarray, mu: float, sigma_w: float, w: int) -> np.ndarray:
    """SNR plane of one boxcar width (debug plane for pin P7)."""
    x, n_dm, n_t, rs = _as_x(x)
    out = np.empty((n_dm, n_t), dtype=np.float64)
    _load().spd_oracle_snr_fixed_width(_p(x), n_dm, n_t, rs, float(mu), float(sigma_w), int(w), _p(out))
    return out


def snr_at(x: np.ndarray, mu: float, sig: np.ndarray, dm, t, w) -> np.ndarray:
    """SNR_w(dm, t) for listed triples, by direct summation."""
    x, n_dm, n_t, rs = _as_x(x)
    sig = np.ascontiguousarray(sig, dtype=np.float64)
    dm = np.ascontiguousarray(dm, dtype=np.int64)
    t = np.ascontiguousarray(t, dtype=np.int64)
    w = np.ascontiguousarray(w, dtype=np.int32)
    out = np.empty(dm.size, dtype=np.float64)
    _load().spd_oracle_snr_at(_p(x), n_t, rs, float(mu), _p(sig), sig.size, _p(dm), _p(t), _p(w), dm.size, _p(out))
    return out


def candidates(snr: np.ndarray, width: np.ndarray, f_T: float):
    """O4: every sample with SNR >= f_T -> (dm, t, snr, width) arrays in (dm, t) order."""
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    width = np.ascontiguousarray(width, dtype=np.int32)
    n_dm, n_t = snr.shape
    L = _load()
    cnt = L.spd_oracle_candidates(_p(snr), _p(width), n_dm, n_t, float(f_T), 0, None, None, None, None)
    c_dm = np.empty(cnt, dtype=np.int64); c_t = np.empty(cnt, dtype=np.int64)
    c_snr = np.empty(cnt, dtype=np.float64); c_w = np.empty(cnt, dtype=np.int32)
    L.spd_oracle_candidates(_p(snr), _p(width), n_dm, n_t, float(f_T), cnt, _p(c_dm), _p(c_t), _p(c_snr), _p(c_w))
    return c_dm, c_t, c_snr, c_w


def stats_rows(x: np.ndarray, nmax_for_sigma: int = 0):
    """One Stats per DM row: O1 (and O1b) on one row at a time (reading A3's per-row alternative)."""
    return [full_stats(x[d:d + 1], nmax_for_sigma) for d in range(x.shape[0])]


def sweep_rows(x: np.ndarray, row_stats, nmax: int, mode):
    """O3r: Algorithm 1 with the statistics of each row: returns (snr f64, width i32, margin f64, sig f64 [n_dm][nmax])."""
    x, n_dm, n_t, rs = _as_x(x)
    mu = np.ascontiguousarray([s.mean for s in row_stats], dtype=np.float64)
    sig = np.ascontiguousarray([sigma_table(s.sigma, s.sigma_nmax, nmax, mode) for s in row_stats], dtype=np.float64)
    snr = np.empty((n_dm, n_t), dtype=np.float64)
    width = np.empty((n_dm, n_t), dtype=np.int32)
    margin = np.empty((n_dm, n_t), dtype=np.float64)
    _load().spd_oracle_sweep_rows(_p(x), n_dm, n_t, rs, _p(mu), _p(sig), int(nmax), _p(snr), _p(width), _p(margin))
    return snr, width, margin, sig


def decimated_levels(w0: int, levels: int):
    """Width grid of O5: [(level, decimation 2^l, smallest w', largest w')]; Nmax = w0 * 2^(levels-1)."""
    assert w0 >= 2 and w0 % 2 == 0 and levels >= 1
    return [(l, 1 << l, 1 if l == 0 else w0 // 2 + 1, w0) for l in range(levels)]


def sweep_decimated(x: np.ndarray, mu: float, sigma: float, sig_nmax: float, mode, w0: int, levels: int):
    """O5 (reading A20): decimation in time + boxcar.  Returns one dict per level:
    {level, D, x (float64 decimated rows), snr, width (effective, 0 = no width fits), margin, sig (sigma_N, N = 1..w0*D)}.
    sigma_N is that of the exhaustive search of the SAME Nmax = w0 * 2^(levels-1) (eq. 4 / eq. 5 / anchored)."""
    x, n_dm, n_t, rs = _as_x(x)
    nmax = w0 * (1 << (levels - 1))
    sig_all = sigma_table(sigma, sig_nmax, nmax, mode)
    L = _load()
    cur = np.ascontiguousarray(x[:, :n_t], dtype=np.float64)
    out = []
    for lvl, D, wmin, wmax in decimated_levels(w0, levels):
        if lvl > 0:
            nxt = np.empty((n_dm, cur.shape[1] // 2), dtype=np.float64)
            L.spd_oracle_decimate2(_p(cur), n_dm, cur.shape[1], _p(nxt))
            cur = nxt
        n_l = cur.shape[1]
        snr = np.empty((n_dm, n_l), dtype=np.float64)
        width = np.empty((n_dm, n_l), dtype=np.int32)
        margin = np.empty((n_dm, n_l), dtype=np.float64)
        sig = np.ascontiguousarray(sig_all[: w0 * D])
        if n_l > 0:
            L.spd_oracle_sweep_level(_p(cur), n_dm, n_l, float(mu), _p(sig), int(w0), int(wmin), int(lvl), _p(snr), _p(width), _p(margin))
        out.append(dict(level=lvl, D=D, x=cur, snr=snr, width=width, margin=margin, sig=sig))
    return out


def candidates_decimated(levels, f_T: float):
    """O4 over the levels of O5 (PAPER.md:87-93 applied to every level plane of reading A20): every level position with
    SNR >= f_T -> one record (dm, t = i 2^l in the ORIGINAL series, snr, effective width N, level), level by level in
    (dm, i) order.  A pulse is usually reported by several levels: nothing is merged (a plain list)."""
    dm, t, snr, w, lv = [], [], [], [], []
    for L in levels:
        c_dm, c_i, c_snr, c_w = candidates(L["snr"], L["width"], f_T)
        dm.append(c_dm); t.append(c_i * int(L["D"])); snr.append(c_snr); w.append(c_w)
        lv.append(np.full(c_dm.size, int(L["level"]), dtype=np.int32))
    return (np.concatenate(dm), np.concatenate(t), np.concatenate(snr), np.concatenate(w), np.concatenate(lv))


def search_decimated(x: np.ndarray, w0: int, levels: int, mode="sqrt", f_T: float = 6.0):
    """The decimated path O1 -> O1b -> O2 -> O5 -> O4 on one array (Nmax = w0 * 2^(levels-1)); returns a dict."""
    m = _MODES[mode]
    nmax = w0 * (1 << (levels - 1))
    st = full_stats(x, nmax if m != 0 else 0)
    lv = sweep_decimated(x, st.mean, st.sigma, st.sigma_nmax, m, w0, levels)
    return dict(stats=st, levels=lv, cand=candidates_decimated(lv, f_T), sig=sigma_table(st.sigma, st.sigma_nmax, nmax, m))


def search(x: np.ndarray, nmax: int, mode="sqrt", f_T: float = 6.0):
    """The whole path O1 -> O1b -> O2 -> O3 -> O4 on one array; returns a dict."""
    m = _MODES[mode]
    st = full_stats(x, nmax if m != 0 else 0)
    sig = sigma_table(st.sigma, st.sigma_nmax, nmax, m)
    snr, width, margin = sweep(x, st.mean, sig)
    cand = candidates(snr, width, f_T)
    return dict(stats=st, sig=sig, snr=snr, width=width, margin=margin, cand=cand)


def set_num_threads(n: int) -> None:
    """OpenMP thread count of the following sweeps (bench.py's per-core figure); no arithmetic is affected."""
    _load()
    C.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def num_threads() -> int:
    """Threads the OpenMP sweep will use (reported as cpu_baseline.cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1
