"""ctypes wrapper around oracle/trd_oracle.cpp -- ORACLE, TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2003_03174_b200 (the seeded inputs are
passed in as plain numpy arrays and a plain dict of cuts).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "trd_oracle.cpp")
_LIB = os.path.join(_HERE, "build", "libtrd_oracle.so")
_lib = None

N_LAYERS_MAX = 6
PION_MASS = 0.13957                                # GeV: the mass hypothesis of the material corrections [R33]
REFIT_VAR = (1.0, 25.0, 2.5e-3, 2.5e-3, 0.25)     # default reset variances of the TRD-only refit [R31]


class OrcConfig(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_stacks", C.c_int32), ("n_layers", C.c_int32), ("n_hyp", C.c_int32),
        ("layer_x", C.c_double * N_LAYERS_MAX),
        ("z_max", C.c_double), ("pad_length", C.c_double), ("bz_tesla", C.c_double),
        ("sigma_y", C.c_double), ("sigma_z", C.c_double), ("sigma_dydx", C.c_double),
        ("n_sigma_road", C.c_double), ("n_sigma_angle", C.c_double),
        ("chi2_cut", C.c_double), ("chi2_penalty", C.c_double), ("max_snp", C.c_double),
        ("sy_c0", C.c_double), ("sy_c2", C.c_double), ("sd_c0", C.c_double), ("sd_c2", C.c_double),
        ("sin_lorentz", C.c_double), ("tan_tilt", C.c_double), ("res_model", C.c_int32), ("pad_", C.c_int32),
        ("x_ref", C.c_double), ("refit_var", C.c_double * 5),
        ("x_over_x0", C.c_double), ("eloss", C.c_double), ("eloss_fluct", C.c_double), ("mass", C.c_double),
        ("bz_r2", C.c_double), ("bz_z2", C.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Returns the path of the shared library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        os.makedirs(os.path.dirname(_LIB), exist_ok=True)
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        assert _lib.orc_sizeof_config() == C.sizeof(OrcConfig)
        _lib.orc_update.restype = C.c_double
    return _lib


def make_config(cfg: dict) -> OrcConfig:
    c = OrcConfig()
    for k in ("n_sectors", "n_stacks", "n_layers", "n_hyp"):
        setattr(c, k, int(cfg[k]))
    for i, v in enumerate(cfg["layer_x"]):
        c.layer_x[i] = float(v)
    for k in ("z_max", "pad_length", "bz_tesla", "sigma_y", "sigma_z", "sigma_dydx", "n_sigma_road",
              "n_sigma_angle", "chi2_cut", "chi2_penalty", "max_snp"):
        setattr(c, k, float(cfg[k]))
    # measurement model of PAPER.md:62, 66 (absent keys = the constant model of the configs)
    for k in ("sy_c0", "sy_c2", "sd_c0", "sd_c2", "sin_lorentz", "tan_tilt"):
        setattr(c, k, float(cfg.get(k, 0.0)))
    c.res_model = int(cfg.get("res_model", 0))
    c.x_ref = float(cfg.get("x_ref", 247.0))
    for i, v in enumerate(cfg.get("refit_var", REFIT_VAR)):
        c.refit_var[i] = float(v)
    # material in front of every layer [R32, R33]; absent = none
    for k in ("x_over_x0", "eloss", "eloss_fluct"):
        setattr(c, k, float(cfg.get(k, 0.0)))
    c.mass = float(cfg.get("mass", PION_MASS))
    # field inhomogeneity Bz(r, z) = bz (1 + bz_r2 r^2 + bz_z2 z^2) [R35]; absent = uniform
    c.bz_r2 = float(cfg.get("bz_r2", 0.0)); c.bz_z2 = float(cfg.get("bz_z2", 0.0))
    return c


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def tri_to_full(c15):
    c15 = np.asarray(c15, float)
    m = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            m[i, j] = m[j, i] = c15[k]
            k += 1
    return m


def full_to_tri(m):
    return np.array([m[i, j] for i in range(5) for j in range(i + 1)], float)


def propagate(cfg: dict, p, c15, x, x_new, want_jacobian=False):
    """In-frame helix propagation.  Returns (ok, p, c15, x[, F])."""
    p = np.array(p, float); c15 = np.array(c15, float); xx = C.c_double(x)
    F = np.zeros((5, 5))
    ok = lib().orc_propagate(C.byref(make_config(cfg)), _dp(p), _dp(c15), C.byref(xx), C.c_double(x_new), _dp(F))
    out = (bool(ok), p, c15, xx.value)
    return out + (F,) if want_jacobian else out


def rotate(cfg: dict, p, c15, x, beta, want_jacobian=False):
    p = np.array(p, float); c15 = np.array(c15, float); xx = C.c_double(x)
    J = np.zeros((5, 5))
    ok = lib().orc_rotate(C.byref(make_config(cfg)), _dp(p), _dp(c15), C.byref(xx), C.c_double(beta), _dp(J))
    out = (bool(ok), p, c15, xx.value)
    return out + (J,) if want_jacobian else out


def propagate_to_layer(cfg: dict, p, c15, x, sector, x_layer):
    p = np.array(p, float); c15 = np.array(c15, float); xx = C.c_double(x); sec = C.c_int32(sector)
    ok = lib().orc_propagate_to_layer(C.byref(make_config(cfg)), _dp(p), _dp(c15), C.byref(xx), C.byref(sec),
                                      C.c_double(x_layer))
    return bool(ok), p, c15, xx.value, sec.value


def update(cfg: dict, p, c15, ym, zm, layer: int = 0):
    p = np.array(p, float); c15 = np.array(c15, float)
    chi2 = lib().orc_update(C.byref(make_config(cfg)), _dp(p), _dp(c15), C.c_double(ym), C.c_double(zm), int(layer))
    return p, c15, float(chi2)


def material(cfg: dict, p, c15, direction: int = 1):
    """One slab of material at the current point (direction +1 outward, -1 inward).  Returns (ok, p, c15)."""
    p = np.array(p, float); c15 = np.array(c15, float)
    ok = lib().orc_material(C.byref(make_config(cfg)), _dp(p), _dp(c15), int(direction))
    return bool(ok), p, c15


def road(cfg: dict, p, c15, layer: int = 0):
    p = np.array(p, float); c15 = np.array(c15, float); out = np.zeros(6)
    lib().orc_road(C.byref(make_config(cfg)), _dp(p), _dp(c15), _dp(out), int(layer))
    return dict(road_y=out[0], road_z=out[1], tanphi=out[2], Sinv=np.array([[out[3], out[4]], [out[4], out[5]]]))


def candidates(cfg: dict, tl: dict, p, c15, sector: int, layer: int, brute: bool = False, cap: int = 4096,
               chamber_dx=None):
    """Accepted candidates (caller's tracklet index, chi2 increment) of one state at one layer."""
    y, z, d, ch = (np.ascontiguousarray(tl[k]) for k in ("tl_y", "tl_z", "tl_dydx", "tl_chamber"))
    p = np.array(p, float); c15 = np.array(c15, float)
    oi = np.zeros(cap, np.int32); oc = np.zeros(cap)
    n = lib().orc_candidates(C.byref(make_config(cfg)), _fp(y), _fp(z), _fp(d), _ip(ch), C.c_int64(y.shape[0]),
                             _dp(p), _dp(c15), int(sector), int(layer), int(brute), _ip(oi), _dp(oc), cap,
                             _dp(np.ascontiguousarray(chamber_dx, np.float64)) if chamber_dx is not None else None)
    assert n <= cap
    return oi[:n].copy(), oc[:n].copy()


def match(cfg: dict, data: dict, brute: bool = False, n_threads: int = 0, lo: int = 0,
          hi: Optional[int] = None, count_distinct: bool = False) -> dict:
    """The whole tracking step on tracks [lo, hi) of `data` against all its tracklets.

    `data` holds the float32 arrays of paper_2003_03174_b200.workloads.generate (or any dict with the
    same keys).  Returns SoA outputs in double plus per-track n_evals and fragility margin, the
    operation counters and the two wall times.
    """
    y, z, d, ch = (np.ascontiguousarray(data[k]) for k in ("tl_y", "tl_z", "tl_dydx", "tl_chamber"))
    assert y.dtype == np.float32 and ch.dtype == np.int32
    hi = data["x"].shape[0] if hi is None else hi
    par = np.ascontiguousarray(data["par"][:, lo:hi]); cov = np.ascontiguousarray(data["cov"][:, lo:hi])
    x = np.ascontiguousarray(data["x"][lo:hi]); sec = np.ascontiguousarray(data["sector"][lo:hi])
    assert par.dtype == np.float32 and cov.dtype == np.float32 and sec.dtype == np.int32
    n = x.shape[0]
    out = dict(idx=np.zeros((6, n), np.int32), par=np.zeros((5, n)), cov=np.zeros((15, n)), x=np.zeros(n),
               sector=np.zeros(n, np.int32), chi2=np.zeros(n), n_matched=np.zeros(n, np.int32),
               n_evals=np.zeros(n, np.int32), margin=np.zeros(n))
    counters = np.zeros(6, np.int64); seconds = np.zeros(2)
    # time-frame association: interaction ids of tracklets and tracks, if the inputs carry them
    n_ia = int(data.get("n_interactions", 0) or 0)
    if n_ia > 1:
        tl_ia = np.ascontiguousarray(data["tl_interaction"]); trk_ia = np.ascontiguousarray(data["interaction"][lo:hi])
        assert tl_ia.dtype == np.int32 and trk_ia.dtype == np.int32
        ia_args = (_ip(tl_ia), _ip(trk_ia), n_ia)
    else:
        ia_args = (None, None, 1)
    # radial chamber offsets for the two-stage propagation, float64 per chamber, if given
    dx = data.get("chamber_dx")
    if dx is not None:
        dx = np.ascontiguousarray(dx, np.float64)
        assert dx.shape[0] == cfg["n_sectors"] * cfg["n_stacks"] * cfg["n_layers"]
    touched = np.zeros(y.shape[0], np.uint8) if count_distinct else None
    rc = lib().orc_match(C.byref(make_config(cfg)), _fp(y), _fp(z), _fp(d), _ip(ch), C.c_int64(y.shape[0]),
                         _fp(par), _fp(cov), _fp(x), _ip(sec), C.c_int64(n), int(brute), int(n_threads),
                         _ip(out["idx"]), _dp(out["par"]), _dp(out["cov"]), _dp(out["x"]), _ip(out["sector"]),
                         _dp(out["chi2"]), _ip(out["n_matched"]), _ip(out["n_evals"]), _dp(out["margin"]),
                         counters.ctypes.data_as(C.POINTER(C.c_int64)), _dp(seconds), *ia_args,
                         _dp(dx) if dx is not None else None,
                         touched.ctypes.data_as(C.POINTER(C.c_ubyte)) if touched is not None else None)
    if rc != 0:
        raise RuntimeError(f"orc_match failed: {rc}")
    out["counters"] = dict(zip(("n_prop", "n_rot", "n_road", "n_cand", "n_upd", "n_scanned"), counters.tolist()))
    out["seconds"] = dict(index=float(seconds[0]), match=float(seconds[1]))
    if touched is not None:
        out["counters"]["n_distinct_cand"] = int(touched.sum())     # distinct tracklets inside some road
    return out


def match_alternatives(cfg: dict, data: dict, tracks, target_idx, eps: float = 1e-4, max_runs: int = 256) -> dict:
    """Is the chain `target_idx[:, k]` a legitimate result for track `tracks[k]`?

    The track is replayed with the decisions closer than `eps` (relative) to their threshold taken either way, until the
    target chain comes out or `max_runs` replays are spent.  Returns `found` (number of replays, negative = not found)
    and the outputs of the replay that reached the target, all with one column per selected track."""
    y, z, d, ch = (np.ascontiguousarray(data[k]) for k in ("tl_y", "tl_z", "tl_dydx", "tl_chamber"))
    par = np.ascontiguousarray(data["par"]); cov = np.ascontiguousarray(data["cov"])
    x = np.ascontiguousarray(data["x"]); sec = np.ascontiguousarray(data["sector"])
    assert par.dtype == np.float32 and cov.dtype == np.float32 and sec.dtype == np.int32
    sel = np.ascontiguousarray(tracks, np.int64)
    tgt = np.ascontiguousarray(target_idx, np.int32)
    k = sel.shape[0]
    assert tgt.shape == (6, k)
    out = dict(found=np.zeros(k, np.int32), idx=np.zeros((6, k), np.int32), par=np.zeros((5, k)), cov=np.zeros((15, k)),
               x=np.zeros(k), sector=np.zeros(k, np.int32), chi2=np.zeros(k), n_matched=np.zeros(k, np.int32),
               n_evals=np.zeros(k, np.int32))
    if k == 0:
        return out
    n_ia = int(data.get("n_interactions", 0) or 0)
    if n_ia > 1:
        tl_ia = np.ascontiguousarray(data["tl_interaction"]); trk_ia = np.ascontiguousarray(data["interaction"])
        ia_args = (_ip(tl_ia), _ip(trk_ia), n_ia)
    else:
        ia_args = (None, None, 1)
    dx = data.get("chamber_dx")
    if dx is not None:
        dx = np.ascontiguousarray(dx, np.float64)
    rc = lib().orc_match_alternatives(
        C.byref(make_config(cfg)), _fp(y), _fp(z), _fp(d), _ip(ch), C.c_int64(y.shape[0]), _fp(par), _fp(cov), _fp(x),
        _ip(sec), C.c_int64(x.shape[0]), sel.ctypes.data_as(C.POINTER(C.c_int64)), C.c_int64(k), _ip(tgt),
        C.c_double(eps), int(max_runs), _ip(out["found"]), _ip(out["idx"]), _dp(out["par"]), _dp(out["cov"]),
        _dp(out["x"]), _ip(out["sector"]), _dp(out["chi2"]), _ip(out["n_matched"]), _ip(out["n_evals"]), *ia_args,
        _dp(dx) if dx is not None else None)
    if rc != 0:
        raise RuntimeError(f"orc_match_alternatives failed: {rc}")
    return out


def refit(cfg: dict, data: dict, matched: dict, min_tracklets: int = 2) -> dict:
    """TRD-only inward refit of the chains in `matched` (the dict returned by match, or the CUDA path's output widened
    to float64) to the plane x_ref.  Returns par, cov, x, sector, chi2, n_used."""
    y, z, ch = (np.ascontiguousarray(data[k]) for k in ("tl_y", "tl_z", "tl_chamber"))
    n = matched["x"].shape[0]
    idx = np.ascontiguousarray(matched["idx"], np.int32)
    par = np.ascontiguousarray(matched["par"], np.float64); cov = np.ascontiguousarray(matched["cov"], np.float64)
    x = np.ascontiguousarray(matched["x"], np.float64); sec = np.ascontiguousarray(matched["sector"], np.int32)
    dx = data.get("chamber_dx")
    if dx is not None:
        dx = np.ascontiguousarray(dx, np.float64)
    out = dict(par=np.zeros((5, n)), cov=np.zeros((15, n)), x=np.zeros(n), sector=np.zeros(n, np.int32),
               chi2=np.zeros(n), n_used=np.zeros(n, np.int32))
    rc = lib().orc_refit(C.byref(make_config(cfg)), _fp(y), _fp(z), _ip(ch), C.c_int64(y.shape[0]),
                         _dp(dx) if dx is not None else None, _ip(idx), _dp(par), _dp(cov), _dp(x), _ip(sec), C.c_int64(n),
                         int(min_tracklets), _dp(out["par"]), _dp(out["cov"]), _dp(out["x"]), _ip(out["sector"]),
                         _dp(out["chi2"]), _ip(out["n_used"]))
    if rc != 0:
        raise RuntimeError(f"orc_refit failed: {rc}")
    return out


def max_threads() -> int:
    return int(lib().orc_max_threads())
