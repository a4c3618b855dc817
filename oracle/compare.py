"""Comparator: GPU results vs the oracle under BASELINE.json:north_star's tolerances.

TEST INFRASTRUCTURE (same import rule as spd_oracle.py).  Pure numpy on arrays the caller
hands in; the "GPU" side arrives as plain numpy arrays, nothing here imports the CUDA path.

Rules (SURVEY.md §8(c) "Comparator"):
  mu          |d| <= 1e-6 * max(|mu|, sigma)
  sigma       |d| <= 1e-6 * sigma           (sigma_Nmax likewise)
  SNR         every sample |d| <= max(1e-3, 1e-4 * |snr_oracle|)
  width       equal wherever the oracle's margin (best - second best) > 1e-3; elsewhere the GPU's
              width must be one whose oracle SNR (direct summation) is within 1e-3 of the best
  candidates  equal as SETS of (dm, t) after dropping, from both sides, samples whose oracle SNR
              is within 1e-3 of the threshold; matched records obey the SNR / width rules
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

from . import spd_oracle as O

SNR_ABS = 1e-3
SNR_REL = 1e-4
TIE = 1e-3
STAT_REL = 1e-6


@dataclass
class Report:
    ok: bool = True
    msgs: list = field(default_factory=list)
    info: Dict[str, float] = field(default_factory=dict)

    def fail(self, m: str):
        self.ok = False
        self.msgs.append(m)

    def __bool__(self):
        return self.ok

    def __str__(self):
        return ("OK " if self.ok else "FAIL ") + "; ".join(self.msgs) + " " + str(self.info)


def compare_stats(g_mean: float, g_sigma: float, o: O.Stats, g_sigma_nmax: Optional[float] = None) -> Report:
    r = Report()
    tol_mu = STAT_REL * max(abs(o.mean), o.sigma)
    r.info["d_mean"] = abs(g_mean - o.mean)
    r.info["d_sigma_rel"] = abs(g_sigma - o.sigma) / o.sigma
    if not abs(g_mean - o.mean) <= tol_mu:
        r.fail(f"mean {g_mean!r} vs {o.mean!r} (tol {tol_mu:.3g})")
    if not abs(g_sigma - o.sigma) <= STAT_REL * o.sigma:
        r.fail(f"sigma {g_sigma!r} vs {o.sigma!r}")
    if g_sigma_nmax is not None:
        r.info["d_sigma_nmax_rel"] = abs(g_sigma_nmax - o.sigma_nmax) / o.sigma_nmax
        if not abs(g_sigma_nmax - o.sigma_nmax) <= STAT_REL * o.sigma_nmax:
            r.fail(f"sigma_nmax {g_sigma_nmax!r} vs {o.sigma_nmax!r}")
    return r


def compare_planes(x: np.ndarray, mu: float, sig: np.ndarray,
                   g_snr: np.ndarray, g_width: np.ndarray,
                   o_snr: np.ndarray, o_width: np.ndarray, o_margin: np.ndarray,
                   dm_offset_rows: Optional[np.ndarray] = None) -> Report:
    """x is the float32 input the ORACLE planes were computed from (rows aligned with the planes)."""
    r = Report()
    g_snr = np.asarray(g_snr, dtype=np.float64)
    g_width = np.asarray(g_width).astype(np.int64)
    if g_snr.shape != o_snr.shape or g_width.shape != o_width.shape:
        r.fail(f"shape {g_snr.shape}/{g_width.shape} vs {o_snr.shape}")
        return r
    if not np.all(np.isfinite(g_snr)):
        r.fail(f"{np.count_nonzero(~np.isfinite(g_snr))} non-finite GPU SNR values")
        return r
    d = np.abs(g_snr - o_snr)
    tol = np.maximum(SNR_ABS, SNR_REL * np.abs(o_snr))
    bad = d > tol
    r.info["snr_max_abs_err"] = float(d.max()) if d.size else 0.0
    r.info["snr_violations"] = int(bad.sum())
    if bad.any():
        i = np.argwhere(bad)[0]
        r.fail(f"SNR: {int(bad.sum())} samples out of tolerance, first at {tuple(i)}: "
               f"{g_snr[tuple(i)]!r} vs {o_snr[tuple(i)]!r}")
    mism = g_width != o_width
    r.info["width_mismatch"] = int(mism.sum())
    hard = mism & (o_margin > TIE)
    if hard.any():
        i = np.argwhere(hard)[0]
        r.fail(f"width: {int(hard.sum())} mismatches outside near-ties, first at {tuple(i)}: "
               f"{int(g_width[tuple(i)])} vs {int(o_width[tuple(i)])} (margin {o_margin[tuple(i)]:.3g})")
    soft = mism & ~(o_margin > TIE)
    r.info["width_near_tie_exempt"] = int(soft.sum())
    r.info["near_tie_rate"] = float(np.count_nonzero(~(o_margin > TIE))) / max(1, o_margin.size)
    if soft.any():
        idx = np.argwhere(soft)
        s_at = O.snr_at(x, mu, sig, idx[:, 0], idx[:, 1], g_width[soft].astype(np.int32))
        best = o_snr[soft]
        worse = ~(np.abs(s_at - best) <= TIE)   # NaN (width that does not fit) counts as a failure
        if worse.any():
            k = int(np.argmax(worse))
            r.fail(f"width: {int(worse.sum())} near-tie widths whose oracle SNR is not within {TIE} of best, "
                   f"first at {tuple(idx[k])}: width {int(g_width[soft][k])} snr {s_at[k]!r} vs best {best[k]!r}")
    return r


def compare_planes_level(x: np.ndarray, mu: float, sig_all: np.ndarray, w0: int, level: dict,
                         g_snr: np.ndarray, g_width: np.ndarray) -> Report:
    """One level of the decimated search (oracle O5, `level` = one dict of spd_oracle.sweep_decimated) against the GPU's
    plane of that level.  Same rules as compare_planes; in addition a position where none of the level's widths fits must
    be (-inf, 0) on both sides, and a width reported inside a near-tie must lie on the level's grid (a multiple of
    D = 2^l with w0/2 < N/D <= w0, or 1 <= N <= w0 at level 0) and is re-summed over the ORIGINAL samples x."""
    r = Report()
    D, lvl = int(level["D"]), int(level["level"])
    o_snr, o_width, o_margin = level["snr"], level["width"], level["margin"]
    g_snr = np.asarray(g_snr, dtype=np.float64)
    g_width = np.asarray(g_width).astype(np.int64)
    if g_snr.shape != o_snr.shape or g_width.shape != o_width.shape:
        r.fail(f"shape {g_snr.shape}/{g_width.shape} vs {o_snr.shape}")
        return r
    none = o_width == 0
    if np.any(g_width[none] != 0) or np.any(g_snr[none] != -np.inf):
        r.fail(f"{int(np.count_nonzero((g_width != 0) & none))} positions where no width of the level fits are not (-inf, 0)")
    ok = ~none
    if np.any(g_width[ok] == 0) or not np.all(np.isfinite(g_snr[ok])):
        r.fail("GPU reports no width / a non-finite SNR where the level has widths that fit")
        return r
    d = np.abs(g_snr[ok] - o_snr[ok])
    bad = d > np.maximum(SNR_ABS, SNR_REL * np.abs(o_snr[ok]))
    r.info["snr_max_abs_err"] = float(d.max()) if d.size else 0.0
    r.info["snr_violations"] = int(bad.sum())
    if bad.any():
        r.fail(f"level {lvl} SNR: {int(bad.sum())} samples out of tolerance")
    mism = ok & (g_width != o_width)
    hard = mism & (o_margin > TIE)
    r.info["width_mismatch"] = int(mism.sum())
    if hard.any():
        i = np.argwhere(hard)[0]
        r.fail(f"level {lvl} width: {int(hard.sum())} mismatches outside near-ties, first at {tuple(i)}: "
               f"{int(g_width[tuple(i)])} vs {int(o_width[tuple(i)])}")
    soft = mism & ~(o_margin > TIE)
    r.info["width_near_tie_exempt"] = int(soft.sum())
    r.info["near_tie_rate"] = float(np.count_nonzero(ok & ~(o_margin > TIE))) / max(1, int(ok.sum()))
    if soft.any():
        idx = np.argwhere(soft)
        N = g_width[soft]
        wp = N // D
        on_grid = (N % D == 0) & (wp <= w0) & (wp >= (1 if lvl == 0 else w0 // 2 + 1)) & (idx[:, 1] + wp <= o_snr.shape[1])
        s_at = O.snr_at(x, mu, sig_all, idx[:, 0], idx[:, 1] * D, N.astype(np.int32))
        worse = ~on_grid | ~(np.abs(s_at - o_snr[soft]) <= TIE)
        if worse.any():
            k = int(np.argmax(worse))
            r.fail(f"level {lvl} width: {int(worse.sum())} near-tie widths off the grid or not within {TIE} of best, first at "
                   f"{tuple(idx[k])}: width {int(N[k])}")
    return r


def compare_candidates(g_dm, g_t, g_snr, g_width, g_count: int, capacity: int,
                       o_snr: np.ndarray, o_width: np.ndarray, o_margin: np.ndarray,
                       f_T: float, x: np.ndarray, mu: float, sig: np.ndarray) -> Report:
    """GPU list (unordered) vs the brute filter of the oracle planes, as sets of (dm, t).

    x, mu, sig are the float32 input, mean and sigma_w table the ORACLE planes were computed from (rows aligned with
    the planes): a record whose width differs from the oracle's inside a near-tie is re-summed with them (snr_at), the
    same validity rule compare_planes applies (SURVEY.md 8(c) "Comparator": "elsewhere the GPU width must be one whose
    oracle SNR is within 1e-3 of best")."""
    r = Report()
    n_dm, n_t = o_snr.shape
    g_dm = np.asarray(g_dm).astype(np.int64); g_t = np.asarray(g_t).astype(np.int64)
    g_snr = np.asarray(g_snr, dtype=np.float64); g_width = np.asarray(g_width).astype(np.int64)
    if g_count > capacity:
        r.fail(f"overflow: count {g_count} > capacity {capacity} (comparison needs the whole list)")
        return r
    if g_dm.size != g_count:
        r.fail(f"list length {g_dm.size} != count {g_count}")
        return r
    if g_count and (g_dm.min() < 0 or g_dm.max() >= n_dm or g_t.min() < 0 or g_t.max() >= n_t):
        r.fail("candidate index out of range")
        return r
    gkey = g_dm * n_t + g_t
    if np.unique(gkey).size != gkey.size:
        r.fail("duplicate (dm, t) records in the GPU list")
    near = np.abs(o_snr - f_T) <= TIE
    okey_all = np.flatnonzero((o_snr >= f_T).ravel())
    near_flat = near.ravel()
    okey = okey_all[~near_flat[okey_all]]
    gkeep = ~near_flat[gkey]
    r.info["oracle_hits"] = int(okey_all.size)
    r.info["gpu_hits"] = int(g_count)
    r.info["near_threshold_exempt"] = int(near.sum())
    gk = np.sort(gkey[gkeep])
    if gk.size != okey.size or not np.array_equal(gk, okey):
        missing = np.setdiff1d(okey, gk); extra = np.setdiff1d(gk, okey)
        r.fail(f"candidate sets differ: {missing.size} missing, {extra.size} extra "
               f"(first missing {divmod(int(missing[0]), n_t) if missing.size else None}, "
               f"first extra {divmod(int(extra[0]), n_t) if extra.size else None})")
        return r
    # matched records: SNR and width rules
    os_ = o_snr.ravel()[gkey]; ow = o_width.ravel()[gkey]
    d = np.abs(g_snr - os_)
    bad = d > np.maximum(SNR_ABS, SNR_REL * np.abs(os_))
    if bad.any():
        r.fail(f"{int(bad.sum())} candidate SNRs out of tolerance")
    mism = g_width != ow
    marg = o_margin.ravel()[gkey]
    hard = mism & (marg > TIE)
    if hard.any():
        r.fail(f"{int(hard.sum())} candidate widths differ outside near-ties")
    soft = mism & ~(marg > TIE)
    r.info["width_near_tie_exempt"] = int(soft.sum())
    if soft.any():
        s_at = O.snr_at(x, mu, sig, g_dm[soft], g_t[soft], g_width[soft].astype(np.int32))
        worse = ~(np.abs(s_at - os_[soft]) <= TIE)   # NaN (a width that does not fit the row or exceeds nmax) fails
        if worse.any():
            k = int(np.argmax(worse))
            r.fail(f"{int(worse.sum())} near-tie candidate widths whose oracle SNR is not within {TIE} of best, first at "
                   f"({int(g_dm[soft][k])}, {int(g_t[soft][k])}): width {int(g_width[soft][k])} snr {s_at[k]!r} vs {os_[soft][k]!r}")
    return r


def level_of_width(N: np.ndarray, w0: int, levels: int) -> np.ndarray:
    """Level of the decimated search a reported EFFECTIVE width belongs to (-1: not on the grid).  The grids of the
    levels are disjoint: 1..w0 at level 0, then D (w0/2 + 1) .. D w0 in steps of D = 2^l."""
    N = np.asarray(N).astype(np.int64)
    out = np.full(N.shape, -1, dtype=np.int64)
    out[(N >= 1) & (N <= w0)] = 0
    for l in range(1, levels):
        D = 1 << l
        out[(N % D == 0) & (N // D > w0 // 2) & (N // D <= w0) & (out < 0)] = l
    return out


def compare_candidates_decimated(g_dm, g_t, g_snr, g_width, g_count: int, capacity: int, levels, w0: int, f_T: float,
                                 x: np.ndarray, mu: float, sig_all: np.ndarray) -> Report:
    """GPU list of a decimated search (unordered; record.t in the ORIGINAL series, record.width = effective width) vs the
    brute filter of every level plane of oracle O5 (`levels` = spd_oracle.sweep_decimated).  A record belongs to the
    level its width lies on; per level the rules are compare_candidates': equal as sets of (dm, i = t / 2^l) outside 1e-3 of
    the threshold, SNR within tolerance, width equal outside near-ties and otherwise on the level's grid, fitting the row
    and with an oracle SNR (re-summed over the original samples) within 1e-3 of best."""
    r = Report()
    g_dm = np.asarray(g_dm).astype(np.int64); g_t = np.asarray(g_t).astype(np.int64)
    g_snr = np.asarray(g_snr, dtype=np.float64); g_width = np.asarray(g_width).astype(np.int64)
    if g_count > capacity:
        r.fail(f"overflow: count {g_count} > capacity {capacity} (comparison needs the whole list)")
        return r
    if g_dm.size != g_count:
        r.fail(f"list length {g_dm.size} != count {g_count}")
        return r
    lv_of = level_of_width(g_width, w0, len(levels))
    if np.any(lv_of < 0):
        r.fail(f"{int(np.count_nonzero(lv_of < 0))} records whose width is on no level's grid")
        return r
    r.info.update(oracle_hits=0, gpu_hits=int(g_count), near_threshold_exempt=0, width_near_tie_exempt=0)
    for L in levels:
        lvl, D = int(L["level"]), int(L["D"])
        o_snr, o_width, o_margin = L["snr"], L["width"], L["margin"]
        n_dm, n_l = o_snr.shape
        sel = lv_of == lvl
        dm, t, sn, wd = g_dm[sel], g_t[sel], g_snr[sel], g_width[sel]
        if np.any(t % D != 0):
            r.fail(f"level {lvl}: record.t is not a multiple of {D}")
            return r
        i = t // D
        if dm.size and (dm.min() < 0 or dm.max() >= n_dm or i.min() < 0 or i.max() >= max(n_l, 1) or n_l == 0):
            r.fail(f"level {lvl}: candidate index out of range")
            return r
        gkey = dm * max(n_l, 1) + i
        if np.unique(gkey).size != gkey.size:
            r.fail(f"level {lvl}: duplicate (dm, t) records")
        near = np.abs(o_snr - f_T) <= TIE
        okey_all = np.flatnonzero((o_snr >= f_T).ravel())
        near_flat = near.ravel()
        okey = okey_all[~near_flat[okey_all]]
        gk = np.sort(gkey[~near_flat[gkey]])
        r.info["oracle_hits"] += int(okey_all.size)
        r.info["near_threshold_exempt"] += int(near.sum())
        if gk.size != okey.size or not np.array_equal(gk, okey):
            missing = np.setdiff1d(okey, gk); extra = np.setdiff1d(gk, okey)
            r.fail(f"level {lvl}: candidate sets differ: {missing.size} missing, {extra.size} extra")
            return r
        os_ = o_snr.ravel()[gkey]; ow = o_width.ravel()[gkey]; marg = o_margin.ravel()[gkey]
        bad = np.abs(sn - os_) > np.maximum(SNR_ABS, SNR_REL * np.abs(os_))
        if bad.any():
            r.fail(f"level {lvl}: {int(bad.sum())} candidate SNRs out of tolerance")
        mism = wd != ow
        hard = mism & (marg > TIE)
        if hard.any():
            r.fail(f"level {lvl}: {int(hard.sum())} candidate widths differ outside near-ties")
        soft = mism & ~(marg > TIE)
        r.info["width_near_tie_exempt"] += int(soft.sum())
        if soft.any():
            fits = i[soft] + wd[soft] // D <= n_l
            s_at = O.snr_at(x, mu, sig_all, dm[soft], t[soft], wd[soft].astype(np.int32))
            worse = ~fits | ~(np.abs(s_at - os_[soft]) <= TIE)
            if worse.any():
                r.fail(f"level {lvl}: {int(worse.sum())} near-tie candidate widths that do not fit or are not within {TIE} of best")
    return r

