"""Thin ctypes binding of libctr.so (include/ctr.h): argument marshalling only.

Every function has the name of the C entry point it calls and takes torch CUDA tensors (fp32,
contiguous) purely as device memory; the stream is torch's current stream. Nothing is computed
here and there is no fallback: if libctr.so is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

_LIB_PATH = Path(__file__).resolve().parent / "libctr.so"
_lib = None

CTR_OK, CTR_EINVAL, CTR_EGEOM, CTR_ENOMEM, CTR_ECUDA, CTR_EARCH, CTR_ETOOBIG = 0, -1, -2, -3, -4, -5, -6


class CtrError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        msg = f"{where}: {_strerror(status)} ({status})"
        if detail:
            msg += f": {detail}"
        super().__init__(msg)


class ctr_geometry(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_float), ("dy", C.c_float), ("dz", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("cz", C.c_float),
                ("nviews", C.c_int32), ("theta0", C.c_float), ("dtheta", C.c_float),
                ("angles", C.POINTER(C.c_float)),
                ("nu", C.c_int32), ("nv", C.c_int32), ("du", C.c_float), ("dv", C.c_float),
                ("u_off", C.c_float), ("v_off", C.c_float), ("dso", C.c_float), ("dsd", C.c_float),
                ("det_type", C.c_int32), ("batch", C.c_int32), ("flags", C.c_int32)]


CTR_GEOM_NO_TABLES = 1
CTR_GEOM_NO_GRAPHS = 2
CTR_GEOM_NO_STORED_P = 4
CTR_GEOM_NO_LAZY_CGLS = 8


class ctr_params(C.Structure):
    _fields_ = [("n_outer", C.c_int32), ("n_cgls", C.c_int32), ("n_gd", C.c_int32),
                ("lam", C.c_float), ("sigma_quantile", C.c_float), ("eps", C.c_float),
                ("armijo_t0", C.c_float), ("armijo_rho", C.c_float), ("armijo_c", C.c_float),
                ("armijo_max", C.c_int32), ("weights_mode", C.c_int32), ("positivity", C.c_int32),
                ("warm_start", C.c_int32), ("fidelity_mode", C.c_int32), ("p1_step", C.c_float),
                ("backprojector", C.c_int32)]


class ctr_sweep_stat(C.Structure):
    _fields_ = [("sigma", C.c_double), ("e0", C.c_double), ("g2", C.c_double),
                ("k", C.c_int32), ("pad", C.c_int32)]


class ctr_peaks(C.Structure):
    _fields_ = [("fma_tflops", C.c_double), ("fma2_tflops", C.c_double), ("issue_gwinst", C.c_double), ("mixed_gwinst", C.c_double),
                ("l1_tbs", C.c_double), ("smem_tbs", C.c_double), ("l2_tbs", C.c_double), ("hbm_copy_gbs", C.c_double),
                ("sm_count", C.c_int32), ("pad", C.c_int32)]


EXPORTS = ["ctr_default_params", "ctr_create", "ctr_destroy", "ctr_forward", "ctr_back", "ctr_back_pixel", "ctr_cgls",
           "ctr_update_weights", "ctr_eptv_step", "ctr_reconstruct", "ctr_reconstruct_w",
           "ctr_set_params", "ctr_get_stats", "ctr_launch_count", "ctr_strerror", "ctr_last_error",
           "ctr_profile_enable", "ctr_profile_read", "ctr_measure_peaks", "ctr_path_info", "ctr_forward_noalloc"]


def load_library():
    """dlopen libctr.so (built in tree by paper_1009_2288_b200.build). Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise FileNotFoundError(f"{_LIB_PATH} is missing: run `python -m paper_1009_2288_b200.build` "
                                "(there is no CPU or PyTorch fallback)")
    L = C.CDLL(str(_LIB_PATH))
    H, vp, fp = C.c_void_p, C.c_void_p, C.c_void_p
    L.ctr_default_params.argtypes = [C.POINTER(ctr_params)]
    L.ctr_default_params.restype = None
    L.ctr_create.argtypes = [C.POINTER(ctr_geometry), C.POINTER(H)]
    L.ctr_destroy.argtypes = [H]
    L.ctr_destroy.restype = None
    L.ctr_forward.argtypes = [H, fp, fp, vp]
    L.ctr_back.argtypes = [H, fp, fp, vp]
    L.ctr_forward_noalloc.argtypes = [C.POINTER(ctr_geometry), fp, fp, vp]
    L.ctr_back_pixel.argtypes = [H, fp, fp, vp]
    L.ctr_cgls.argtypes = [H, fp, fp, C.c_int, vp]
    L.ctr_update_weights.argtypes = [H, fp, fp, C.c_float, fp, vp]
    L.ctr_eptv_step.argtypes = [H, fp, fp, fp, C.c_float, vp]
    L.ctr_reconstruct.argtypes = [H, fp, fp, C.POINTER(ctr_params), vp]
    L.ctr_reconstruct_w.argtypes = [H, fp, fp, fp, C.POINTER(ctr_params), vp]
    L.ctr_set_params.argtypes = [H, C.POINTER(ctr_params)]
    L.ctr_get_stats.argtypes = [H, C.POINTER(ctr_sweep_stat), C.c_size_t]
    L.ctr_profile_enable.argtypes = [H, C.c_int]
    L.ctr_profile_read.argtypes = [H, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.ctr_measure_peaks.argtypes = [C.POINTER(ctr_peaks), C.c_int]
    L.ctr_launch_count.argtypes = [H]
    L.ctr_launch_count.restype = C.c_longlong
    L.ctr_strerror.argtypes = [C.c_int]
    L.ctr_strerror.restype = C.c_char_p
    L.ctr_last_error.argtypes = [H]
    L.ctr_last_error.restype = C.c_char_p
    L.ctr_path_info.argtypes = [H]
    L.ctr_path_info.restype = C.c_char_p
    _lib = L
    return L


def _strerror(status: int) -> str:
    try:
        return load_library().ctr_strerror(status).decode()
    except Exception:
        return "error"


def make_geometry(g) -> ctr_geometry:
    """g: a dict with ctr_geometry field names or an object with .geometry_dict()."""
    d = g.geometry_dict() if hasattr(g, "geometry_dict") else dict(g)
    cg = ctr_geometry()
    defaults = dict(ndim=2, nz=1, nv=1, dz=1.0, dv=1.0, cx=0.0, cy=0.0, cz=0.0, theta0=0.0, dtheta=0.0,
                    u_off=0.0, v_off=0.0, det_type=0, batch=1, flags=0)
    defaults.update({k: v for k, v in d.items() if k != "angles"})
    for name, ctype in ctr_geometry._fields_:
        if name == "angles":
            continue
        setattr(cg, name, defaults[name])
    ang = d.get("angles")
    if ang is not None:
        arr = (C.c_float * len(ang))(*[float(a) for a in ang])
        cg._angles_keepalive = arr
        cg.angles = C.cast(arr, C.POINTER(C.c_float))
    return cg


def make_params(p=None, **over) -> ctr_params:
    cp = ctr_params()
    load_library().ctr_default_params(C.byref(cp))
    d = {}
    if p is not None:
        d.update(p.params_dict() if hasattr(p, "params_dict") else dict(p))
    d.update(over)
    if "lambda" in d:
        d["lam"] = d.pop("lambda")
    names = {n for n, _ in ctr_params._fields_}
    for k, v in d.items():
        if k not in names:
            raise KeyError(f"unknown ctr_params field {k!r}")
        setattr(cp, k, v)
    return cp


def _ptr(t: torch.Tensor, n_expected: int | None = None, name: str = "tensor"):
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous fp32 CUDA tensor")
    if n_expected is not None and t.numel() != n_expected:
        raise ValueError(f"{name}: expected {n_expected} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Handle:
    """Owns a ctr_handle*. Methods mirror the C entry points one to one."""

    def __init__(self, geometry, flags: int = 0):
        self._L = load_library()
        self.geom = make_geometry(geometry)
        self.geom.flags |= int(flags)
        self._h = C.c_void_p()
        rc = self._L.ctr_create(C.byref(self.geom), C.byref(self._h))
        if rc != CTR_OK:
            self._h = C.c_void_p()
            raise CtrError(rc, "ctr_create")
        g = self.geom
        self.n_img = g.batch * g.nx * g.ny * g.nz
        self.n_sino = g.batch * g.nviews * g.nu * g.nv
        self.img_shape = (g.nz, g.ny, g.nx) if g.ndim == 3 else (g.batch, g.ny, g.nx)
        self.sino_shape = (g.nviews, g.nv, g.nu) if g.ndim == 3 else (g.batch, g.nviews, g.nu)
        self.w_shape = (g.ndim,) + self.img_shape

    def _check(self, rc, where):
        if rc != CTR_OK:
            raise CtrError(rc, where, self._L.ctr_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.ctr_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def ctr_forward(self, img, sino):
        self._check(self._L.ctr_forward(self._h, _ptr(img, self.n_img, "img"), _ptr(sino, self.n_sino, "sino"), _stream()), "ctr_forward")
        return sino

    def ctr_back(self, sino, img):
        self._check(self._L.ctr_back(self._h, _ptr(sino, self.n_sino, "sino"), _ptr(img, self.n_img, "img"), _stream()), "ctr_back")
        return img

    def ctr_back_pixel(self, sino, img):
        self._check(self._L.ctr_back_pixel(self._h, _ptr(sino, self.n_sino, "sino"), _ptr(img, self.n_img, "img"), _stream()), "ctr_back_pixel")
        return img

    def ctr_cgls(self, b, x, n_iter):
        self._check(self._L.ctr_cgls(self._h, _ptr(b, self.n_sino, "b"), _ptr(x, self.n_img, "x"), int(n_iter), _stream()), "ctr_cgls")
        return x

    def ctr_update_weights(self, x, w, quantile=0.90, sigma=None):
        sp = _ptr(sigma, self.geom.batch, "sigma") if sigma is not None else C.c_void_p()
        self._check(self._L.ctr_update_weights(self._h, _ptr(x, self.n_img, "x"), _ptr(w, self.n_img * self.geom.ndim, "w"),
                                               C.c_float(quantile), sp, _stream()), "ctr_update_weights")
        return w

    def ctr_eptv_step(self, x, v, w, lam):
        self._check(self._L.ctr_eptv_step(self._h, _ptr(x, self.n_img, "x"), _ptr(v, self.n_img, "v"),
                                          _ptr(w, self.n_img * self.geom.ndim, "w"), C.c_float(lam), _stream()), "ctr_eptv_step")
        return x

    def ctr_reconstruct(self, sino, img, params=None, w=None):
        pp = C.byref(params) if params is not None else None
        wp = _ptr(w, self.n_img * self.geom.ndim, "w") if w is not None else C.c_void_p()
        self._check(self._L.ctr_reconstruct_w(self._h, _ptr(sino, self.n_sino, "sino"), _ptr(img, self.n_img, "img"),
                                              wp, pp, _stream()), "ctr_reconstruct")
        return img

    def ctr_set_params(self, params):
        self._check(self._L.ctr_set_params(self._h, C.byref(params)), "ctr_set_params")

    def ctr_get_stats(self):
        """Synchronises; returns a list of dicts ordered [sweep][slice]."""
        n = self._L.ctr_get_stats(self._h, None, 0)
        if n < 0:
            self._check(n, "ctr_get_stats")
        buf = (ctr_sweep_stat * max(n, 1))()
        n2 = self._L.ctr_get_stats(self._h, buf, n)
        if n2 < 0:
            self._check(n2, "ctr_get_stats")
        return [dict(sigma=buf[i].sigma, e0=buf[i].e0, g2=buf[i].g2, k=buf[i].k) for i in range(n)]

    def ctr_profile_enable(self, on: bool):
        self._check(self._L.ctr_profile_enable(self._h, int(bool(on))), "ctr_profile_enable")

    def ctr_profile_read(self):
        """Synchronises; returns {kind: (milliseconds, intervals)} for the handle's own launches."""
        ms = (C.c_double * 5)()
        cnt = (C.c_longlong * 5)()
        self._check(self._L.ctr_profile_read(self._h, ms, cnt), "ctr_profile_read")
        kinds = ["forward", "back", "vector", "tv", "layout"]
        return {k: (ms[i], int(cnt[i])) for i, k in enumerate(kinds)}

    def ctr_path_info(self) -> dict:
        return dict(kv.split("=", 1) for kv in self._L.ctr_path_info(self._h).decode().split(";") if kv)

    def ctr_launch_count(self) -> int:
        return int(self._L.ctr_launch_count(self._h))


def ctr_measure_peaks(reps: int = 5) -> dict:
    """Synchronous microbenchmarks on the current device (include/ctr.h); returns the ctr_peaks fields."""
    pk = ctr_peaks()
    rc = load_library().ctr_measure_peaks(C.byref(pk), int(reps))
    if rc != CTR_OK:
        raise CtrError(rc, "ctr_measure_peaks")
    return {n: getattr(pk, n) for n, _ in ctr_peaks._fields_ if n != "pad"}


def ctr_forward_noalloc(geometry, img: torch.Tensor, sino: torch.Tensor) -> torch.Tensor:
    """sino = P img for one 2D slice without a handle and without any allocation (include/ctr.h: fixed scratch,
    CTR_ETOOBIG beyond 512 x 512 pixels / 65536 rays / 4096 views; overlapping calls race)."""
    L = load_library()
    cg = make_geometry(geometry)
    n_img, n_sino = cg.nx * cg.ny, cg.nviews * cg.nu
    rc = L.ctr_forward_noalloc(C.byref(cg), _ptr(img, n_img, "img"), _ptr(sino, n_sino, "sino"), _stream())
    if rc != CTR_OK:
        raise CtrError(rc, "ctr_forward_noalloc")
    return sino


def ctr_create(geometry, flags: int = 0) -> Handle:
    """flags: ctr_geometry.flags bits (CTR_GEOM_NO_TABLES) OR-ed into the geometry."""
    return Handle(geometry, flags)


def ctr_destroy(h: Handle) -> None:
    h.close()
