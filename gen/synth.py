"""Row-addressable seeded generator for the five BASELINE.json workloads.

Recipe: every row d of config c is drawn from
``numpy.random.Generator(PCG64(SeedSequence([SEED0, c, d])))`` so that any row can be
regenerated alone (the oracle works on row subsets of the big configs without the whole
array).  The pulse list comes from ``SeedSequence([SEED0, c, 999999])``.  Amplitudes use
the NOMINAL sigma of the config.  Output is float32, row-major, time fastest.

The paper (§3) evaluates on unspecified "SKA-like data"; these synthetic
arrays take that shape (about 6000 DM trials, 64 us sampling) and stand in for it.

Nothing here is part of the detection method: no mean/sigma, boxcar, SNR or threshold
arithmetic lives in this module.
"""
from __future__ import annotations

import math
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

SEED0 = 16110970  # arXiv number of the paper, used as the root seed
_PULSE_STREAM = 999999

# best-boxcar response of a unit-peak Gaussian of given FWHM is 0.8186*sqrt(FWHM)*peak
# (generator convention for config 3 -- not from the paper)
_GAUSS_BOXCAR_RESPONSE = 0.8186


@dataclass(frozen=True)
class Pulse:
    row: int          # DM-trial index of the pulse centre row
    start: int        # first sample (rect) or centre sample (gauss)
    width: int        # width in samples (rect) or FWHM (gauss)
    amp: float        # per-sample amplitude (rect) or peak amplitude (gauss)
    snr: float        # target boxcar SNR at the best width (nan if not defined)
    kind: str         # "rect" | "gauss"


@dataclass(frozen=True)
class Config:
    cid: int
    name: str
    n_dm: int
    n_t: int
    mu: float = 0.0
    sigma: float = 1.0
    drift_amp: float = 0.0        # sinusoidal baseline amplitude (config 4)
    drift_period: int = 65536
    pulse_kind: str = "rect"      # "rect_fixed" | "rect_snr" | "gauss_snr" | "rect_amp" | "rect_log" | "none"
    n_pulses: int = 0
    nmax: Tuple[int, ...] = (32,)
    sigma_mode: str = "sqrt"      # "sqrt" = eq. 4, "linear" = eq. 5
    threshold: float = 6.0
    dm_smear: int = 0             # pulse copied to rows d +- k, k <= dm_smear, amplitude *(1-|k|/(dm_smear+1))
    t_samp: float = 64e-6         # seconds per sample
    extra_pulses: Tuple[Pulse, ...] = field(default_factory=tuple)

    @property
    def n(self) -> int:
        return self.n_dm * self.n_t


CONFIGS: Dict[int, Config] = {
    1: Config(1, "C1-small", 64, 16384, pulse_kind="rect_fixed", n_pulses=5, nmax=(32,), threshold=6.0),
    2: Config(2, "C2-offset", 1024, 131072, mu=100.0, sigma=20.0, pulse_kind="rect_snr", n_pulses=50,
              nmax=(64,), threshold=6.0),
    3: Config(3, "C3-SKA-like", 6000, 262144, pulse_kind="gauss_snr", n_pulses=200, nmax=(128,),
              threshold=7.0, dm_smear=3),
    4: Config(4, "C4-signal-dominated", 2048, 262144, drift_amp=0.5, pulse_kind="rect_amp", n_pulses=500,
              nmax=(512,), sigma_mode="linear", threshold=6.0),
    5: Config(5, "C5-width-sweep", 4096, 524288, pulse_kind="rect_log", n_pulses=1000,
              nmax=(8, 32, 128, 512), threshold=6.0),
}


def get_config(cid: int) -> Config:
    return CONFIGS[int(cid)]


def custom_config(n_dm: int, n_t: int, *, cid: int = 1000, **kw) -> Config:
    """A free-form config for tests (same seeding scheme, user-chosen id)."""
    base = Config(cid, kw.pop("name", f"custom-{cid}"), n_dm, n_t, pulse_kind=kw.pop("pulse_kind", "none"))
    return replace(base, **kw)


def _row_rng(cfg: Config, row: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED0, cfg.cid, int(row)])))


def pulse_table(cfg: Config) -> List[Pulse]:
    """The injected-pulse truth table of a config (deterministic)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED0, cfg.cid, _PULSE_STREAM])))
    out: List[Pulse] = []
    k = cfg.pulse_kind
    n = cfg.n_pulses
    if k == "none" or n == 0:
        pass
    elif k == "rect_fixed":      # C1: widths 1,2,4,8,16, SNR 10
        widths = [1, 2, 4, 8, 16][:n]
        for w in widths:
            row = int(rng.integers(0, cfg.n_dm))
            start = int(rng.integers(0, cfg.n_t - w + 1))
            out.append(Pulse(row, start, w, 10.0 * cfg.sigma / math.sqrt(w), 10.0, "rect"))
    elif k == "rect_snr":        # C2: W~U{1..64}, S~U(7,20)
        wmax = min(64, cfg.n_t)
        for _ in range(n):
            w = int(rng.integers(1, wmax + 1))
            s = float(rng.uniform(7.0, 20.0))
            row = int(rng.integers(0, cfg.n_dm))
            start = int(rng.integers(0, cfg.n_t - w + 1))
            out.append(Pulse(row, start, w, s * cfg.sigma / math.sqrt(w), s, "rect"))
    elif k == "gauss_snr":       # C3: FWHM~U{1..128}, S~U(6,30)
        for _ in range(n):
            fwhm = int(rng.integers(1, 129))
            s = float(rng.uniform(6.0, 30.0))
            row = int(rng.integers(0, cfg.n_dm))
            centre = int(rng.integers(0, cfg.n_t))
            amp = s * cfg.sigma / (_GAUSS_BOXCAR_RESPONSE * math.sqrt(fwhm))
            out.append(Pulse(row, centre, fwhm, amp, s, "gauss"))
    elif k == "rect_amp":        # C4: W~U{100..500}, per-sample amplitude ~U(3,10) sigma
        wlo, whi = 100, min(500, cfg.n_t)
        for _ in range(n):
            w = int(rng.integers(min(wlo, whi), whi + 1))
            a = float(rng.uniform(3.0, 10.0))
            row = int(rng.integers(0, cfg.n_dm))
            start = int(rng.integers(0, cfg.n_t - w + 1))
            out.append(Pulse(row, start, w, a * cfg.sigma, a * math.sqrt(w), "rect"))
    elif k == "rect_log":        # C5: W log-uniform 1..512, S~U(6,50)
        wmax = min(512, cfg.n_t)
        for _ in range(n):
            w = int(min(wmax, max(1, round(math.exp(rng.uniform(0.0, math.log(wmax)))))))
            s = float(rng.uniform(6.0, 50.0))
            row = int(rng.integers(0, cfg.n_dm))
            start = int(rng.integers(0, cfg.n_t - w + 1))
            out.append(Pulse(row, start, w, s * cfg.sigma / math.sqrt(w), s, "rect"))
    else:
        raise ValueError(f"unknown pulse_kind {k!r}")
    out.extend(cfg.extra_pulses)
    return out


def _pulse_profile(p: Pulse, n_t: int) -> Tuple[int, np.ndarray]:
    """(first sample, float64 profile) of one pulse clipped to [0, n_t)."""
    if p.kind == "rect":
        lo, hi = max(0, p.start), min(n_t, p.start + p.width)
        return lo, np.full(max(0, hi - lo), p.amp, dtype=np.float64)
    if p.kind == "gauss":
        half = 3 * p.width + 1
        lo, hi = max(0, p.start - half), min(n_t, p.start + half + 1)
        t = np.arange(lo, hi, dtype=np.float64)
        prof = p.amp * np.exp(-4.0 * math.log(2.0) * ((t - p.start) / float(p.width)) ** 2)
        return lo, prof
    raise ValueError(p.kind)


def _row_pulse_index(cfg: Config) -> Dict[int, List[Tuple[int, np.ndarray]]]:
    idx: Dict[int, List[Tuple[int, np.ndarray]]] = {}
    for p in pulse_table(cfg):
        lo, prof = _pulse_profile(p, cfg.n_t)
        for k in range(-cfg.dm_smear, cfg.dm_smear + 1):
            r = p.row + k
            if 0 <= r < cfg.n_dm:
                scale = 1.0 - abs(k) / float(cfg.dm_smear + 1)
                idx.setdefault(r, []).append((lo, prof * scale))
    return idx


def pulse_rows(cfg: Config) -> List[int]:
    """Sorted rows that carry any injected signal."""
    return sorted(_row_pulse_index(cfg).keys())


def _fill_row(cfg: Config, row: int, out: np.ndarray, pidx) -> None:
    rng = _row_rng(cfg, row)
    phase = float(rng.uniform(0.0, 2.0 * math.pi))  # always drawn so the noise stream is config-independent
    rng.standard_normal(out.shape[0], dtype=np.float32, out=out)
    if cfg.sigma != 1.0:
        out *= np.float32(cfg.sigma)
    if cfg.mu != 0.0:
        out += np.float32(cfg.mu)
    if cfg.drift_amp != 0.0:
        t = np.arange(cfg.n_t, dtype=np.float64)
        out += (cfg.drift_amp * cfg.sigma * np.sin(2.0 * math.pi * t / cfg.drift_period + phase)).astype(np.float32)
    for lo, prof in pidx.get(row, ()):
        out[lo:lo + prof.shape[0]] += prof.astype(np.float32)


def make_rows(cfg: Config, rows: Sequence[int]) -> np.ndarray:
    """float32 [len(rows)][n_t]: the listed rows of the config's array, regenerated alone."""
    pidx = _row_pulse_index(cfg)
    out = np.empty((len(rows), cfg.n_t), dtype=np.float32)
    for i, r in enumerate(rows):
        _fill_row(cfg, int(r), out[i], pidx)
    return out


def make_array(cfg: Config, out: Optional[np.ndarray] = None, threads: Optional[int] = None,
               row_lo: int = 0, row_hi: Optional[int] = None) -> np.ndarray:
    """float32 [row_hi-row_lo][n_t]: rows row_lo..row_hi-1 of the config's array (default: all rows).

    ``out`` may be any writable float32 2-D array of that shape (e.g. a view of a pinned torch
    tensor).  Rows are filled by a thread pool; the result does not depend on the thread count.
    """
    row_hi = cfg.n_dm if row_hi is None else row_hi
    nrows = row_hi - row_lo
    if out is None:
        out = np.empty((nrows, cfg.n_t), dtype=np.float32)
    assert out.shape == (nrows, cfg.n_t) and out.dtype == np.float32
    pidx = _row_pulse_index(cfg)
    threads = threads or min(32, os.cpu_count() or 1)

    def work(block):
        for r in block:
            _fill_row(cfg, r, out[r - row_lo], pidx)

    blocks = [range(b, min(b + 16, row_hi)) for b in range(row_lo, row_hi, 16)]
    if threads <= 1 or len(blocks) <= 1:
        for b in blocks:
            work(b)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(work, blocks))
    return out
