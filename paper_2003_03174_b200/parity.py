"""Element-by-element comparison of two results of the tracking step (plain numpy dicts).

Holds none of the method's arithmetic and imports neither the CUDA binding nor the oracle: the
caller passes `got` (the CUDA path's output) and `want` (the reference result, which also carries
the per-track fragility `margin`).  Criteria (BASELINE.json north_star):

  assignment  tracklet index identical per track and layer, except on tracks whose reference
              margin (smallest relative distance of any discrete decision from its threshold,
              rank gaps included) is below `eps_margin`;
  parameters  |got - want| <= 1e-4 |want| or <= 1e-5, on tracks with identical assignment;
  chi2        |got - want| <= 1e-3 |want| (+ chi2_atol), same tracks;
  integers    n_matched and sector exact, x equal to the reference x rounded to float32 (the output type), on tracks
              with identical assignment.

A track whose assignment differs (allowed only below `eps_margin`) is not skipped: `compare` lists it in
`flip_tracks`, the caller asks the reference side whether the chain found here is one of the results its algorithm
reaches when the decisions closer than `eps_margin` to their threshold are taken the other way, and
`compare_alternatives` then applies the same numeric criteria against that alternative.
"""
from __future__ import annotations

from typing import Dict

import numpy as np

PAR_RTOL = 1e-4
PAR_ATOL = 1e-5
CHI2_RTOL = 1e-3
EPS_MARGIN = 1e-4


def compare(got: Dict[str, np.ndarray], want: Dict[str, np.ndarray], eps_margin: float = EPS_MARGIN,
            chi2_atol: float = 0.0, cov_rtol: float = 2e-3, x_atol: float = 0.0, par_atol: float = PAR_ATOL) -> dict:
    """x_atol: extra tolerance on the output x (0: it must be the reference x rounded to float32).  par_atol: the
    absolute floor of the parameter tolerance, the north_star's 1e-5."""
    n = want["x"].shape[0]
    same = np.all(got["idx"][:, :n] == want["idx"], axis=0)
    fragile = want["margin"] < eps_margin
    mism = ~same
    rep = dict(n_tracks=int(n), n_assign_mismatch=int(mism.sum()), n_fragile=int(fragile.sum()),
               n_unexplained=int((mism & ~fragile).sum()))
    rep["unexplained_tracks"] = np.nonzero(mism & ~fragile)[0][:20].tolist()
    rep["flip_tracks"] = np.nonzero(mism & fragile)[0]            # to be validated with compare_alternatives
    rep["max_margin_of_mismatch"] = float(want["margin"][mism].max()) if mism.any() else 0.0
    s = same
    gp = got["par"][:, :n].astype(np.float64)
    dp = np.abs(gp - want["par"])
    par_ok = (dp <= PAR_RTOL * np.abs(want["par"])) | (dp <= par_atol)
    bad_par = s & ~np.all(par_ok, axis=0)
    rep["n_par_bad"] = int(bad_par.sum())
    rep["par_bad_tracks"] = np.nonzero(bad_par)[0][:20].tolist()
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(s[None, :], dp / np.maximum(np.abs(want["par"]), PAR_ATOL / PAR_RTOL), 0.0)
    rep["par_max_scaled_err"] = [float(v) for v in rel.max(axis=1)] if n else [0.0] * 5
    dc = np.abs(got["chi2"][:n].astype(np.float64) - want["chi2"])
    bad_chi2 = s & ~(dc <= CHI2_RTOL * np.abs(want["chi2"]) + chi2_atol)
    rep["n_chi2_bad"] = int(bad_chi2.sum())
    rep["chi2_bad_tracks"] = np.nonzero(bad_chi2)[0][:20].tolist()
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(s & (want["chi2"] > 0), dc / np.abs(want["chi2"]), 0.0)
    rep["chi2_max_rel_err"] = float(r.max()) if n else 0.0
    gx = got["x"][:n].astype(np.float64)
    ints_ok = (got["n_matched"][:n] == want["n_matched"]) & (got["sector"][:n] == want["sector"]) & \
              ((gx == want["x"].astype(np.float32).astype(np.float64)) | (np.abs(gx - want["x"]) <= x_atol))
    rep["n_int_bad"] = int((s & ~ints_ok).sum())
    # covariance: scaled by sqrt(C_ii C_jj) of the reference
    tri = [(i, j) for i in range(5) for j in range(i + 1)]
    diag = np.stack([want["cov"][i * (i + 1) // 2 + i] for i in range(5)])
    scale = np.stack([np.sqrt(np.abs(diag[i] * diag[j])) for i, j in tri])
    dcov = np.abs(got["cov"][:, :n].astype(np.float64) - want["cov"])
    with np.errstate(divide="ignore", invalid="ignore"):
        rc = np.where(s[None, :] & (scale > 0), dcov / scale, 0.0)
    rep["cov_max_scaled_err"] = float(rc.max()) if n else 0.0
    rep["n_cov_bad"] = int((rc > cov_rtol).any(axis=0).sum())
    if "n_evals" in got and "n_evals" in want:
        rep["n_evals_got"] = int(got["n_evals"][:n].astype(np.int64).sum())
        rep["n_evals_want"] = int(want["n_evals"].astype(np.int64).sum())
        rep["n_evals_bad"] = int((s & ~fragile & (got["n_evals"][:n] != want["n_evals"])).sum())
    rep["ok"] = (rep["n_unexplained"] == 0 and rep["n_par_bad"] == 0 and rep["n_chi2_bad"] == 0
                 and rep["n_int_bad"] == 0 and rep["n_cov_bad"] == 0)
    return rep


def compare_alternatives(got: Dict[str, np.ndarray], alt: Dict[str, np.ndarray], tracks, chi2_atol: float = 0.0,
                         cov_rtol: float = 2e-3, x_atol: float = 0.0, par_atol: float = PAR_ATOL) -> dict:
    """The flipped tracks of `compare`: `alt` holds, for track tracks[k] in column k, the reference side's result
    with its fragile decisions taken so that the chain of `got` comes out (`alt["found"][k]` > 0 if such a result
    exists).  Every flip must be such an alternative, and parameters, chi2, covariance and integers must agree with
    it under the same criteria as everywhere else."""
    tracks = np.asarray(tracks, np.int64)
    k = tracks.shape[0]
    sub = {key: np.asarray(got[key])[..., tracks] for key in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched")}
    want = dict(alt)
    want["margin"] = np.full(k, np.inf)               # nothing is exempt here: the chains must be identical
    rep = compare(sub, want, chi2_atol=chi2_atol, cov_rtol=cov_rtol, x_atol=x_atol, par_atol=par_atol)
    found = np.asarray(alt["found"]) > 0
    rep["n_flips"] = int(k)
    rep["n_not_an_alternative"] = int((~found).sum())
    rep["not_an_alternative_tracks"] = tracks[~found][:20].tolist()
    rep["max_replays"] = int(np.abs(np.asarray(alt["found"])).max()) if k else 0
    rep["ok"] = bool(rep["ok"] and rep["n_not_an_alternative"] == 0 and rep["n_assign_mismatch"] == 0)
    return rep
