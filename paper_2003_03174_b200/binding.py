"""Thin Python binding of include/trdmatch.h (ctypes): argument marshalling only.

Function names and argument order follow the C ABI.  Device arrays are torch CUDA tensors
(torch is used for device memory and streams, nothing else); the *_host calls take numpy
arrays.  Every step of the path runs in the CUDA kernels of csrc/; there is no CPU fallback:
if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np

from . import build as _build

TRD_MAX_LAYERS = 6
TRD_MAX_HYP = 8
TRD_OK, TRD_E_ARG, TRD_E_CUDA, TRD_E_NOMEM, TRD_E_STATE = 0, -1, -2, -3, -4
_STATUS = {0: "TRD_OK", -1: "TRD_E_ARG", -2: "TRD_E_CUDA", -3: "TRD_E_NOMEM", -4: "TRD_E_STATE"}

EXPORTS = ("trd_version", "trd_create", "trd_destroy", "trd_load_tracklets", "trd_load_tracklets_tf", "trd_set_chamber_dx", "trd_match", "trd_match_static", "trd_refit",
           "trd_load_tracklets_host", "trd_match_host", "trd_match_host_async", "trd_wait_host", "trd_get_index_info", "trd_copy_index",
           "trd_last_error", "trd_device_bytes", "trd_kernel_launches", "trd_last_match_kernel_ms", "trd_match_kernel_ms")

_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)


class TrdConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_sectors", C.c_int32), ("n_stacks", C.c_int32),
                ("n_layers", C.c_int32), ("n_hyp", C.c_int32), ("layer_x", C.c_double * TRD_MAX_LAYERS),
                ("z_max", C.c_double), ("pad_length", C.c_double), ("bz_tesla", C.c_double),
                ("sigma_y", C.c_double), ("sigma_z", C.c_double), ("sigma_dydx", C.c_double),
                ("n_sigma_road", C.c_double), ("n_sigma_angle", C.c_double), ("chi2_cut", C.c_double),
                ("chi2_penalty", C.c_double), ("max_snp", C.c_double), ("ybin_width", C.c_double),
                ("track_binning", C.c_int32), ("res_model", C.c_int32),
                ("sy_c0", C.c_double), ("sy_c2", C.c_double), ("sd_c0", C.c_double), ("sd_c2", C.c_double),
                ("sin_lorentz", C.c_double), ("tan_tilt", C.c_double), ("x_ref", C.c_double),
                ("refit_var", C.c_double * 5),
                ("x_over_x0", C.c_double), ("eloss", C.c_double), ("eloss_fluct", C.c_double), ("mass", C.c_double),
                ("bz_r2", C.c_double), ("bz_z2", C.c_double), ("index_sort", C.c_int32), ("reserved_", C.c_int32)]

REFIT_VAR = (1.0, 25.0, 2.5e-3, 2.5e-3, 0.25)     # default reset variances of trd_refit (R31)


class TrdTracksIn(C.Structure):
    _fields_ = [("par", C.c_void_p * 5), ("cov", C.c_void_p * 15), ("x", C.c_void_p), ("sector", C.c_void_p),
                ("interaction", C.c_void_p)]


class TrdTracksOut(C.Structure):
    _fields_ = [("tracklet_idx", C.c_void_p * TRD_MAX_LAYERS), ("par", C.c_void_p * 5), ("cov", C.c_void_p * 15),
                ("x", C.c_void_p), ("sector", C.c_void_p), ("chi2", C.c_void_p), ("n_matched", C.c_void_p),
                ("n_cand_evals", C.c_void_p)]


class TrdRefitOut(C.Structure):
    _fields_ = [("par", C.c_void_p * 5), ("cov", C.c_void_p * 15), ("x", C.c_void_p), ("sector", C.c_void_p),
                ("chi2", C.c_void_p), ("n_used", C.c_void_p)]


class TrdIndexInfo(C.Structure):
    _fields_ = [("n_tracklets", C.c_int64), ("n_zrows", C.c_int32), ("n_ybins", C.c_int32), ("n_bins", C.c_int64),
                ("ybin_width", C.c_double), ("key_bits", C.c_int32), ("n_passes", C.c_int32),
                ("n_interactions", C.c_int32), ("sort_kind", C.c_int32)]


class TrdError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_STATUS.get(code, code)}: {text}")
        self.code = code


_lib = None


def library_path() -> str:
    return _build.LIB_PATH


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: run `python -m paper_2003_03174_b200.build` "
                               "(the TRD matcher has no CPU fallback)")
        l = C.CDLL(path)
        l.trd_version.restype = C.c_int
        l.trd_create.argtypes = [C.POINTER(TrdConfig), C.POINTER(C.c_void_p)]
        l.trd_destroy.argtypes = [C.c_void_p]
        l.trd_destroy.restype = None
        l.trd_load_tracklets.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        l.trd_load_tracklets_host.argtypes = l.trd_load_tracklets.argtypes
        l.trd_load_tracklets_tf.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                            C.c_int64, C.c_void_p]
        l.trd_set_chamber_dx.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        l.trd_match.argtypes = [C.c_void_p, C.POINTER(TrdTracksIn), C.POINTER(TrdTracksOut), C.c_int64, C.c_void_p]
        l.trd_match_static.argtypes = l.trd_match.argtypes
        l.trd_refit.argtypes = [C.c_void_p, C.POINTER(TrdTracksOut), C.POINTER(TrdRefitOut), C.c_int64, C.c_void_p]
        l.trd_match_host.argtypes = l.trd_match.argtypes
        l.trd_match_host_async.argtypes = l.trd_match.argtypes
        l.trd_wait_host.argtypes = [C.c_void_p, C.c_void_p]
        l.trd_get_index_info.argtypes = [C.c_void_p, C.POINTER(TrdIndexInfo)]
        l.trd_copy_index.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        l.trd_last_error.argtypes = [C.c_void_p]
        l.trd_last_error.restype = C.c_char_p
        l.trd_device_bytes.argtypes = [C.c_void_p]
        l.trd_device_bytes.restype = C.c_int64
        l.trd_kernel_launches.argtypes = [C.c_void_p]
        l.trd_kernel_launches.restype = C.c_int64
        l.trd_last_match_kernel_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        l.trd_match_kernel_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int32]
        _lib = l
    return _lib


def make_config(cfg: dict) -> TrdConfig:
    c = TrdConfig()
    c.struct_size = C.sizeof(TrdConfig)
    for k in ("n_sectors", "n_stacks", "n_layers", "n_hyp"):
        setattr(c, k, int(cfg[k]))
    for i, v in enumerate(cfg["layer_x"]):
        c.layer_x[i] = float(v)
    for k in ("z_max", "pad_length", "bz_tesla", "sigma_y", "sigma_z", "sigma_dydx", "n_sigma_road",
              "n_sigma_angle", "chi2_cut", "chi2_penalty", "max_snp"):
        setattr(c, k, float(cfg[k]))
    c.ybin_width = float(cfg.get("ybin_width", 0.0))
    c.track_binning = int(cfg.get("track_binning", 0))
    c.res_model = int(cfg.get("res_model", 0))
    for k in ("sy_c0", "sy_c2", "sd_c0", "sd_c2", "sin_lorentz", "tan_tilt"):
        setattr(c, k, float(cfg.get(k, 0.0)))
    c.x_ref = float(cfg.get("x_ref", 247.0))
    for i, v in enumerate(cfg.get("refit_var", REFIT_VAR)):
        c.refit_var[i] = float(v)
    for k in ("x_over_x0", "eloss", "eloss_fluct"):
        setattr(c, k, float(cfg.get(k, 0.0)))
    c.mass = float(cfg.get("mass", 0.13957))
    c.bz_r2 = float(cfg.get("bz_r2", 0.0)); c.bz_z2 = float(cfg.get("bz_z2", 0.0))
    c.index_sort = int(cfg.get("index_sort", 0)); c.reserved_ = 0
    return c


def _check(h, rc: int):
    if rc != TRD_OK:
        text = lib().trd_last_error(h).decode() if h else ""
        raise TrdError(rc, text)


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    return getattr(stream, "cuda_stream", stream) or None


# ---- the C ABI, same names -------------------------------------------------------------------
def trd_version() -> int:
    return int(lib().trd_version())


def trd_create(cfg: dict) -> C.c_void_p:
    h = C.c_void_p()
    c = make_config(cfg)
    rc = lib().trd_create(C.byref(c), C.byref(h))
    if rc != TRD_OK:
        raise TrdError(rc, "trd_create (bad config, or no CUDA device: there is no CPU fallback)")
    return h


def trd_destroy(h) -> None:
    lib().trd_destroy(h)


def _dev_ptr(t, dtype, n=None):
    import torch
    want = {"f32": torch.float32, "i32": torch.int32}[dtype]
    if not (t.is_cuda and t.dtype == want and t.is_contiguous()):
        raise TypeError(f"expected a contiguous CUDA {want} tensor")
    if n is not None and t.numel() != n:
        raise ValueError("array length mismatch")
    return t.data_ptr()


def trd_load_tracklets(h, d_y, d_z, d_dydx, d_chamber, n: Optional[int] = None, stream=None) -> None:
    n = d_y.numel() if n is None else n
    _check(h, lib().trd_load_tracklets(h, _dev_ptr(d_y, "f32", n), _dev_ptr(d_z, "f32", n), _dev_ptr(d_dydx, "f32", n),
                                       _dev_ptr(d_chamber, "i32", n), n, _stream(stream)))


def trd_load_tracklets_tf(h, d_y, d_z, d_dydx, d_chamber, d_interaction, n_interactions: int, n: Optional[int] = None,
                          stream=None) -> None:
    """Time-frame variant: tracklets carry interaction ids (int32 CUDA tensor); see include/trdmatch.h."""
    n = d_y.numel() if n is None else n
    _check(h, lib().trd_load_tracklets_tf(h, _dev_ptr(d_y, "f32", n), _dev_ptr(d_z, "f32", n), _dev_ptr(d_dydx, "f32", n),
                                          _dev_ptr(d_chamber, "i32", n), _dev_ptr(d_interaction, "i32", n),
                                          int(n_interactions), n, _stream(stream)))


def trd_set_chamber_dx(h, dx: Optional[np.ndarray], stream=None) -> None:
    """Radial chamber offsets (float32 numpy array, one per chamber) for the two-stage propagation; None clears."""
    if dx is None:
        _check(h, lib().trd_set_chamber_dx(h, None, 0, _stream(stream)))
    else:
        _check(h, lib().trd_set_chamber_dx(h, _host_ptr(dx, np.float32), int(dx.size), _stream(stream)))


def alloc_tracks_out(n: int, device="cuda", with_evals: bool = True) -> Dict[str, "object"]:
    import torch
    out = dict(idx=torch.empty((TRD_MAX_LAYERS, n), dtype=torch.int32, device=device),
               par=torch.empty((5, n), dtype=torch.float32, device=device),
               cov=torch.empty((15, n), dtype=torch.float32, device=device),
               x=torch.empty(n, dtype=torch.float32, device=device),
               sector=torch.empty(n, dtype=torch.int32, device=device),
               chi2=torch.empty(n, dtype=torch.float32, device=device),
               n_matched=torch.empty(n, dtype=torch.int32, device=device))
    if with_evals:
        out["n_evals"] = torch.empty(n, dtype=torch.int32, device=device)
    return out


def _row_ptrs(t, rows, n, dtype):
    _dev_ptr(t, dtype, rows * n)
    base = t.data_ptr()
    return [base + 4 * n * k for k in range(rows)]


def trd_match(h, tracks: dict, out: Optional[dict] = None, n_tracks: Optional[int] = None, stream=None) -> dict:
    """tracks: par (5, n) f32, cov (15, n) f32, x (n,) f32, sector (n,) i32, CUDA tensors (SoA rows).
    out: as returned by alloc_tracks_out (allocated if None)."""
    n = tracks["x"].numel() if n_tracks is None else n_tracks
    if out is None:
        out = alloc_tracks_out(n, device=tracks["x"].device)
    tin, tout = TrdTracksIn(), TrdTracksOut()
    if n > 0:
        tin.par[:] = _row_ptrs(tracks["par"], 5, n, "f32")
        tin.cov[:] = _row_ptrs(tracks["cov"], 15, n, "f32")
        tin.x = _dev_ptr(tracks["x"], "f32", n)
        tin.sector = _dev_ptr(tracks["sector"], "i32", n)
        tin.interaction = _dev_ptr(tracks["interaction"], "i32", n) if "interaction" in tracks else None
        tout.tracklet_idx[:] = _row_ptrs(out["idx"], TRD_MAX_LAYERS, n, "i32")
        tout.par[:] = _row_ptrs(out["par"], 5, n, "f32")
        tout.cov[:] = _row_ptrs(out["cov"], 15, n, "f32")
        tout.x = _dev_ptr(out["x"], "f32", n)
        tout.sector = _dev_ptr(out["sector"], "i32", n)
        tout.chi2 = _dev_ptr(out["chi2"], "f32", n)
        tout.n_matched = _dev_ptr(out["n_matched"], "i32", n)
        tout.n_cand_evals = _dev_ptr(out["n_evals"], "i32", n) if "n_evals" in out else None
    _check(h, lib().trd_match(h, C.byref(tin), C.byref(tout), n, _stream(stream)))
    return out


TRD_STATIC_MAX_TRACKS = 32768          # include/trdmatch.h
TRD_STATIC_SCRATCH_BYTES = 7864576


def trd_match_static(h, tracks: dict, out: dict, n_tracks: Optional[int] = None, stream=None) -> dict:
    """trd_match without any device allocation: the library's scratch is a static device array, `out` must be given
    (this wrapper allocates nothing either).  At most TRD_STATIC_MAX_TRACKS tracks per call; calls that overlap on the
    GPU race on the shared scratch (include/trdmatch.h)."""
    n = tracks["x"].numel() if n_tracks is None else n_tracks
    tin, tout = TrdTracksIn(), TrdTracksOut()
    if n > 0:
        tin.par[:] = _row_ptrs(tracks["par"], 5, n, "f32")
        tin.cov[:] = _row_ptrs(tracks["cov"], 15, n, "f32")
        tin.x = _dev_ptr(tracks["x"], "f32", n)
        tin.sector = _dev_ptr(tracks["sector"], "i32", n)
        tin.interaction = _dev_ptr(tracks["interaction"], "i32", n) if "interaction" in tracks else None
        tout.tracklet_idx[:] = _row_ptrs(out["idx"], TRD_MAX_LAYERS, n, "i32")
        tout.par[:] = _row_ptrs(out["par"], 5, n, "f32")
        tout.cov[:] = _row_ptrs(out["cov"], 15, n, "f32")
        tout.x = _dev_ptr(out["x"], "f32", n)
        tout.sector = _dev_ptr(out["sector"], "i32", n)
        tout.chi2 = _dev_ptr(out["chi2"], "f32", n)
        tout.n_matched = _dev_ptr(out["n_matched"], "i32", n)
        tout.n_cand_evals = _dev_ptr(out["n_evals"], "i32", n) if "n_evals" in out else None
    _check(h, lib().trd_match_static(h, C.byref(tin), C.byref(tout), n, _stream(stream)))
    return out


def trd_refit(h, matched: dict, out: Optional[dict] = None, stream=None) -> dict:
    """TRD-only inward refit of the chains in `matched` (the dict trd_match returned, CUDA tensors) to the plane
    x_ref.  Returns par (5, n), cov (15, n), x, sector, chi2, n_used as CUDA tensors."""
    import torch
    n = matched["x"].numel()
    dev = matched["x"].device
    if out is None:
        out = dict(par=torch.empty((5, n), dtype=torch.float32, device=dev), cov=torch.empty((15, n), dtype=torch.float32, device=dev),
                   x=torch.empty(n, dtype=torch.float32, device=dev), sector=torch.empty(n, dtype=torch.int32, device=dev),
                   chi2=torch.empty(n, dtype=torch.float32, device=dev), n_used=torch.empty(n, dtype=torch.int32, device=dev))
    tm, to = TrdTracksOut(), TrdRefitOut()
    if n > 0:
        tm.tracklet_idx[:] = _row_ptrs(matched["idx"], TRD_MAX_LAYERS, n, "i32")
        tm.par[:] = _row_ptrs(matched["par"], 5, n, "f32")
        tm.cov[:] = _row_ptrs(matched["cov"], 15, n, "f32")
        tm.x = _dev_ptr(matched["x"], "f32", n)
        tm.sector = _dev_ptr(matched["sector"], "i32", n)
        to.par[:] = _row_ptrs(out["par"], 5, n, "f32")
        to.cov[:] = _row_ptrs(out["cov"], 15, n, "f32")
        to.x = _dev_ptr(out["x"], "f32", n)
        to.sector = _dev_ptr(out["sector"], "i32", n)
        to.chi2 = _dev_ptr(out["chi2"], "f32", n)
        to.n_used = _dev_ptr(out["n_used"], "i32", n)
    _check(h, lib().trd_refit(h, C.byref(tm), C.byref(to), n, _stream(stream)))
    return out


def _host_ptr(a: np.ndarray, dtype, n=None):
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]):
        raise TypeError(f"expected a C-contiguous numpy {dtype} array")
    if n is not None and a.size != n:
        raise ValueError("array length mismatch")
    return a.ctypes.data


def trd_load_tracklets_host(h, y, z, dydx, chamber, stream=None) -> None:
    n = y.size
    _check(h, lib().trd_load_tracklets_host(h, _host_ptr(y, np.float32, n), _host_ptr(z, np.float32, n),
                                            _host_ptr(dydx, np.float32, n), _host_ptr(chamber, np.int32, n), n,
                                            _stream(stream)))


def alloc_tracks_out_host(n: int, pinned: bool = False) -> Dict[str, np.ndarray]:
    shapes = dict(idx=((TRD_MAX_LAYERS, n), np.int32), par=((5, n), np.float32), cov=((15, n), np.float32),
                  x=((n,), np.float32), sector=((n,), np.int32), chi2=((n,), np.float32),
                  n_matched=((n,), np.int32), n_evals=((n,), np.int32))
    if not pinned:
        return {k: np.empty(s, d) for k, (s, d) in shapes.items()}
    import torch
    tdt = {np.int32: torch.int32, np.float32: torch.float32}
    keep = {k: torch.empty(s, dtype=tdt[d]).pin_memory() for k, (s, d) in shapes.items()}
    out = {k: t.numpy() for k, t in keep.items()}
    out["_pinned"] = keep
    return out


def trd_wait_host(h, stream=None) -> None:
    _check(h, lib().trd_wait_host(h, _stream(stream)))


def trd_match_host_async(h, tracks: dict, out: Optional[dict] = None, stream=None) -> dict:
    """trd_match_host without the final wait: `out` is valid only after trd_wait_host (pinned arrays overlap)."""
    return trd_match_host(h, tracks, out, stream, _async=True)


def trd_match_host(h, tracks: dict, out: Optional[dict] = None, stream=None, _async: bool = False) -> dict:
    """Same as trd_match with numpy arrays; returns when the results are in `out`."""
    n = tracks["x"].size
    if out is None:
        out = alloc_tracks_out_host(n)
    tin, tout = TrdTracksIn(), TrdTracksOut()
    if n > 0:
        def rows(a, r, dt):
            base = _host_ptr(a, dt, r * n)
            return [base + 4 * n * k for k in range(r)]
        tin.par[:] = rows(tracks["par"], 5, np.float32)
        tin.cov[:] = rows(tracks["cov"], 15, np.float32)
        tin.x = _host_ptr(tracks["x"], np.float32, n)
        tin.sector = _host_ptr(tracks["sector"], np.int32, n)
        tout.tracklet_idx[:] = rows(out["idx"], TRD_MAX_LAYERS, np.int32)
        tout.par[:] = rows(out["par"], 5, np.float32)
        tout.cov[:] = rows(out["cov"], 15, np.float32)
        tout.x = _host_ptr(out["x"], np.float32, n)
        tout.sector = _host_ptr(out["sector"], np.int32, n)
        tout.chi2 = _host_ptr(out["chi2"], np.float32, n)
        tout.n_matched = _host_ptr(out["n_matched"], np.int32, n)
        tout.n_cand_evals = _host_ptr(out["n_evals"], np.int32, n) if "n_evals" in out else None
    fn = lib().trd_match_host_async if _async else lib().trd_match_host
    _check(h, fn(h, C.byref(tin), C.byref(tout), n, _stream(stream)))
    return out


def trd_get_index_info(h) -> dict:
    info = TrdIndexInfo()
    _check(h, lib().trd_get_index_info(h, C.byref(info)))
    return {k: getattr(info, k) for k, _ in TrdIndexInfo._fields_}


def trd_copy_index(h, stream=None) -> dict:
    """Sorted positions, sorted keys and the first-position table as numpy arrays (diagnostics)."""
    info = trd_get_index_info(h)
    n = info["n_tracklets"]
    pos = np.empty(n, np.int32); key = np.empty(n, np.uint32); first = np.empty(info["n_bins"] + 1, np.int32)
    _check(h, lib().trd_copy_index(h, pos.ctypes.data, key.ctypes.data, first.ctypes.data, _stream(stream)))
    info = trd_get_index_info(h)                    # sort_kind is final only now
    return dict(info, sorted_pos=pos, sorted_key=key, bin_first=first)


def trd_device_bytes(h) -> int:
    return int(lib().trd_device_bytes(h))


def trd_kernel_launches(h) -> int:
    return int(lib().trd_kernel_launches(h))


def trd_match_kernel_ms(h, n: int) -> list:
    """Device times [ms] of the match kernel in the n most recent trd_match calls (n <= 64), oldest first."""
    ms = (C.c_float * n)()
    _check(h, lib().trd_match_kernel_ms(h, ms, n))
    return [float(v) for v in ms]


def trd_last_match_kernel_ms(h) -> float:
    ms = C.c_float()
    _check(h, lib().trd_last_match_kernel_ms(h, C.byref(ms)))
    return float(ms.value)


# ---- convenience -----------------------------------------------------------------------------
def to_device(data: dict, device="cuda") -> dict:
    """Upload the arrays of workloads.generate as torch tensors (tracks and tracklets)."""
    import torch
    keys = ("par", "cov", "x", "sector", "tl_y", "tl_z", "tl_dydx", "tl_chamber", "interaction", "tl_interaction")
    return {k: torch.from_numpy(np.ascontiguousarray(data[k])).to(device) for k in keys if k in data}


def to_numpy(out: dict) -> dict:
    return {k: v.cpu().numpy() for k, v in out.items()}
