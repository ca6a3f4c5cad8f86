"""Parity metric between a fitter's output and the fp64 oracle (reading A15).

north_star: relative 1e-4 on track parameters, 1e-3 on covariance elements, 1e-3 on chi2.
A relative error of a component that is legitimately ~0 is undefined, so:
  position   |d| <= 1e-4 * r_last            momentum |d| <= 1e-4 * |p|
  covariance |dC_ij| <= 1e-3 * s_i s_j,  s_i = sqrt(max diagonal of i's 3x3 block)
  chi2       |d| <= 1e-3 * max(chi2, 1)
Diverged tracks (A14: oracle chi2 > ndf + 9 sqrt(2 ndf) or any oracle status bit) are excluded
and counted; they must be < 0.1 % of a config.
Pure numpy bookkeeping: no Kalman arithmetic here.
"""
from __future__ import annotations

import numpy as np

TOL_PAR, TOL_COV, TOL_CHI2 = 1e-4, 1e-3, 1e-3
_TRI = [(i, j) for i in range(6) for j in range(i, 6)]


def dense_from_packed(c21: np.ndarray) -> np.ndarray:
    n = c21.shape[1]
    out = np.empty((n, 6, 6))
    for k, (i, j) in enumerate(_TRI):
        out[:, i, j] = c21[k]
        out[:, j, i] = c21[k]
    return out


def diverged_mask(oracle: dict) -> np.ndarray:
    ndf = np.maximum(2 * oracle["nhits"] - 5, 1).astype(np.float64)
    return (oracle["status"] != 0) | (oracle["chi2"] > ndf + 9.0 * np.sqrt(2.0 * ndf))


def compare_fit(gpu: dict, oracle: dict, r_last: float | np.ndarray, max_diverged_frac: float = 1e-3,
                loosen: dict | None = None, ill: np.ndarray | None = None, max_ill_frac: float = 0.0,
                per_track: bool = False, max_strict_fail_frac: float = 1e-2) -> dict:
    """gpu: par[6][n] f32, cov[21][n] f32, chi2[n], nhits[n], status[n]; oracle: O.fit_tracks dict.
    Returns the worst normalised errors (each must be <= 1 to pass) and raises AssertionError on failure.
    `ill` (optional, bool[n]): tracks an ORACLE-SIDE rule identifies as ill-conditioned (stated by the caller,
    e.g. a candidate that took a hit with oracle chi2 > 15 and kinked by many sigma).  Only those are held to the
    tolerances times `loosen`; every other track is held to the stated tolerances, 1.0.  At most `max_ill_frac`
    of the tracks may be marked.  Without `ill`, `loosen` applies to all tracks (callers that still pass it say
    why)."""
    loosen = loosen or {}
    n = oracle["par"].shape[1]
    bad = diverged_mask(oracle)
    ok = ~bad
    frac = bad.mean() if n else 0.0
    assert frac <= max_diverged_frac, f"diverged fraction {frac:.4%}"
    gp = np.asarray(gpu["par"], dtype=np.float64)[:, :n]
    gc = dense_from_packed(np.asarray(gpu["cov"], dtype=np.float64)[:, :n])
    op, oc = oracle["par"], oracle["cov"]
    r_last = np.broadcast_to(np.asarray(r_last, dtype=np.float64), (n,))
    e_pos = np.max(np.abs(gp[:3] - op[:3]), axis=0) / (TOL_PAR * r_last)
    pabs = np.sqrt((op[3:] ** 2).sum(axis=0))
    e_mom = np.max(np.abs(gp[3:] - op[3:]), axis=0) / (TOL_PAR * pabs)
    d = np.diagonal(oc, axis1=1, axis2=2)
    s = np.sqrt(np.concatenate([np.repeat(d[:, :3].max(axis=1, keepdims=True), 3, 1),
                                np.repeat(d[:, 3:].max(axis=1, keepdims=True), 3, 1)], axis=1))
    scale = s[:, :, None] * s[:, None, :]
    e_cov = (np.abs(gc - oc) / (TOL_COV * scale)).reshape(n, -1).max(axis=1)
    # stricter, element-wise: |dC_ij| <= 1e-3 sqrt(C_ii C_jj) -- on the elements where that scale means something:
    # a covariance transported to a surface has NO variance along the surface normal, so for axis-aligned tracks
    # (and for every track that ends on a disc: C_zz = 0) some C_ii are zero up to rounding and the ratio is
    # undefined; elements whose scale is below 1e-2 of their blocks' scale are left to the block metric above
    dd = np.sqrt(np.clip(d, 0.0, None))
    sc_strict = dd[:, :, None] * dd[:, None, :]
    defined = sc_strict >= 1e-2 * scale
    e_cov_strict = np.where(defined, np.abs(gc - oc) / (TOL_COV * np.where(defined, sc_strict, 1.0)), 0.0).reshape(n, -1).max(axis=1)
    gchi = np.asarray(gpu["chi2"], dtype=np.float64)[:n]
    e_chi = np.abs(gchi - oracle["chi2"]) / (TOL_CHI2 * np.maximum(oracle["chi2"], 1.0))
    res = dict(n=n, n_diverged=int(bad.sum()),
               pos=float(e_pos[ok].max(initial=0)), mom=float(e_mom[ok].max(initial=0)),
               cov=float(e_cov[ok].max(initial=0)), chi2=float(e_chi[ok].max(initial=0)),
               cov_strict_fail_frac=float((e_cov_strict[ok] > 1).mean()) if ok.any() else 0.0,
               mom_p99=float(np.percentile(e_mom[ok], 99)) if ok.any() else 0.0,
               cov_p99=float(np.percentile(e_cov[ok], 99)) if ok.any() else 0.0,
               chi2_p99=float(np.percentile(e_chi[ok], 99)) if ok.any() else 0.0)
    assert np.array_equal(np.asarray(gpu["nhits"])[:n][ok], oracle["nhits"][ok]), "nhits differ"
    assert np.array_equal(np.asarray(gpu["status"])[:n][ok], oracle["status"][ok]), "status differ"
    # the stricter element-wise metric |dC_ij| <= 1e-3 sqrt(C_ii C_jj) is ill-posed on the structurally null
    # direction of axis-aligned tracks (A15), so it is not THE bound -- but the fraction of tracks missing it is held
    assert res["cov_strict_fail_frac"] <= max_strict_fail_frac or loosen.get("cov", 1.0) > 1e6, \
        f"{res['cov_strict_fail_frac']:.2e} of the tracks miss the element-wise covariance metric: {res}"
    errs = dict(pos=e_pos, mom=e_mom, cov=e_cov, chi2=e_chi)
    if per_track:
        res["per_track"] = dict(errs, ok=ok)
    if ill is None:
        for key in ("pos", "mom", "cov", "chi2"):
            assert res[key] <= loosen.get(key, 1.0), f"{key} parity failed: {res}"
        return res
    ill = np.asarray(ill, dtype=bool)[:n]
    res["n_ill"] = int((ill & ok).sum())
    assert res["n_ill"] <= max_ill_frac * max(int(ok.sum()), 1), f"{res['n_ill']} of {int(ok.sum())} tracks marked ill-conditioned"
    for key in ("pos", "mom", "cov", "chi2"):
        e = errs[key]
        res[key + "_clean"] = float(e[ok & ~ill].max(initial=0))
        res[key + "_ill"] = float(e[ok & ill].max(initial=0))
        res["n_ill_over_1_" + key] = int((e[ok & ill] > 1).sum())
        assert res[key + "_clean"] <= 1.0, f"{key} parity failed on the well-conditioned tracks: {res}"
        assert res[key + "_ill"] <= loosen.get(key, 1.0), f"{key} parity failed on the ill-conditioned tracks: {res}"
    return res
