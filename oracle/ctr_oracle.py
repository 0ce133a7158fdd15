"""ctypes front end of oracle/ctr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
legs may import this module.  It never imports paper_1009_2288_b200 (the CUDA path).
All arrays are numpy fp64; images are [nz,ny,nx] (2D: [ny,nx] accepted), sinograms
[nviews,nv,nu] (2D: [nviews,nu] accepted).  A batch is a Python loop over slices.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ctr_oracle.c"
_LIB = _HERE / "libctr_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp oracle/ctr_oracle.c -> oracle/libctr_oracle.so (in tree)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class OrcGeom(C.Structure):
    _fields_ = [("ndim", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("cz", C.c_double),
                ("nviews", C.c_int), ("theta0", C.c_double), ("dtheta", C.c_double),
                ("angles", C.POINTER(C.c_double)),
                ("nu", C.c_int), ("nv", C.c_int), ("du", C.c_double), ("dv", C.c_double),
                ("u_off", C.c_double), ("v_off", C.c_double), ("dso", C.c_double),
                ("dsd", C.c_double), ("det_type", C.c_int)]


class OrcParams(C.Structure):
    _fields_ = [("n_outer", C.c_int), ("n_cgls", C.c_int), ("n_gd", C.c_int),
                ("lam", C.c_double), ("sigma_quantile", C.c_double), ("eps", C.c_double),
                ("armijo_t0", C.c_double), ("armijo_rho", C.c_double), ("armijo_c", C.c_double),
                ("armijo_max", C.c_int), ("weights_mode", C.c_int), ("positivity", C.c_int),
                ("reorth", C.c_int)]


_DP = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        G, P = C.POINTER(OrcGeom), C.POINTER(OrcParams)
        i, d = C.c_int, C.c_double
        L.orc_ray.argtypes = [G, i, i, i, _DP, _DP]
        L.orc_forward.argtypes = [G, _DP, _DP]
        L.orc_back.argtypes = [G, _DP, _DP]
        L.orc_matrix_row.argtypes = [G, i, i, i, _DP]
        L.orc_back_eq11.argtypes = [G, _DP, _DP]
        L.orc_cgls.argtypes = [G, _DP, _DP, i, i]
        L.orc_face_mag2.argtypes = [i, i, i, i, _DP, _DP]
        L.orc_sigma.argtypes = [i, i, i, i, _DP, d, d]
        L.orc_sigma.restype = d
        L.orc_weights.argtypes = [i, i, i, i, _DP, d, i, _DP]
        L.orc_gradient.argtypes = [i, i, i, i, _DP, _DP, _DP, d, d, _DP]
        L.orc_energy.argtypes = [i, i, i, i, _DP, _DP, _DP, d, d]
        L.orc_energy.restype = d
        L.orc_eptv_step.argtypes = [i, i, i, i, _DP, _DP, _DP, d, P, _DP]
        L.orc_eptv_step.restype = i
        L.orc_update_weights.argtypes = [i, i, i, i, _DP, d, d, i, _DP]
        L.orc_update_weights.restype = d
        L.orc_reconstruct.argtypes = [G, _DP, P, _DP, _DP, _DP]
        L.orc_num_threads.restype = i
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _f32(x) -> float:
    """The ABI passes float parameters; the oracle uses the double value of that float."""
    return float(np.float32(x))


def make_geom(g) -> OrcGeom:
    """g: a ctr_inputs.Config or a dict with ctr_geometry field names.  Float fields are taken
    at their fp32 value (what the C ABI receives), then promoted to double."""
    d = g.geometry_dict() if hasattr(g, "geometry_dict") else dict(g)
    og = OrcGeom()
    for k in ("ndim", "nx", "ny", "nz", "nviews", "nu", "nv", "det_type"):
        setattr(og, k, int(d.get(k, {"ndim": 2, "nz": 1, "nv": 1, "det_type": 0}.get(k, 0))))
    for k in ("dx", "dy", "dz", "cx", "cy", "cz", "theta0", "dtheta", "du", "dv", "u_off",
              "v_off", "dso", "dsd"):
        setattr(og, k, _f32(d.get(k, {"dz": 1.0, "dv": 1.0}.get(k, 0.0))))
    ang = d.get("angles")
    if ang is not None:
        arr = np.ascontiguousarray(np.asarray(ang, dtype=np.float32).astype(np.float64))
        og._angles_keepalive = arr
        og.angles = arr.ctypes.data_as(_DP)
    return og


def make_params(p) -> OrcParams:
    d = p.params_dict() if hasattr(p, "params_dict") else dict(p)
    op = OrcParams()
    defaults = dict(n_outer=1, n_cgls=1, n_gd=5, lam=0.01, sigma_quantile=0.90, eps=1e-4,
                    armijo_t0=1e-3, armijo_rho=0.5, armijo_c=0.5, armijo_max=16,
                    weights_mode=0, positivity=1, reorth=1)
    defaults.update(d)
    for k in ("n_outer", "n_cgls", "n_gd", "armijo_max", "weights_mode", "positivity", "reorth"):
        setattr(op, k, int(defaults[k]))
    for k in ("lam", "sigma_quantile", "eps", "armijo_t0", "armijo_rho", "armijo_c"):
        setattr(op, k, _f32(defaults[k]))
    return op


def _p(a):
    return a.ctypes.data_as(_DP)


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _dims(og):
    return og.ndim, og.nx, og.ny, og.nz


def ray(g, k, b, a):
    og = make_geom(g)
    S, D = np.zeros(3), np.zeros(3)
    lib().orc_ray(C.byref(og), k, b, a, _p(S), _p(D))
    return S, D


def forward(g, img):
    og = make_geom(g)
    img = _c64(img)
    assert img.size == og.nx * og.ny * og.nz
    sino = np.zeros((og.nviews, og.nv, og.nu))
    lib().orc_forward(C.byref(og), _p(img), _p(sino))
    return sino[:, 0, :] if og.ndim == 2 else sino


def back(g, sino):
    og = make_geom(g)
    sino = _c64(sino)
    assert sino.size == og.nviews * og.nv * og.nu
    img = np.zeros((og.nz, og.ny, og.nx))
    lib().orc_back(C.byref(og), _p(sino), _p(img))
    return img[0] if og.ndim == 2 else img


def back_eq11(g, sino):
    """NEXT-1: the paper's pixel-driven, interpolating backprojector Eq. (11), 2D."""
    og = make_geom(g)
    assert og.ndim == 2
    sino = _c64(sino)
    assert sino.size == og.nviews * og.nu
    img = np.zeros((og.ny, og.nx))
    lib().orc_back_eq11(C.byref(og), _p(sino), _p(img))
    return img


def matrix(g):
    """Dense system matrix [nrays, nvox] by tracing every ray (tiny geometries only)."""
    og = make_geom(g)
    nvox = og.nx * og.ny * og.nz
    A = np.zeros((og.nviews * og.nv * og.nu, nvox))
    r = 0
    for k in range(og.nviews):
        for b in range(og.nv):
            for a in range(og.nu):
                lib().orc_matrix_row(C.byref(og), k, b, a, _p(A[r]))
                r += 1
    return A


def cgls(g, b, x0, n_iter, reorth=True):
    """O4. reorth=True: reading S24 (gradients re-orthogonalised); False: recurrence as printed."""
    og = make_geom(g)
    b = _c64(b)
    x = _c64(x0).copy()
    lib().orc_cgls(C.byref(og), _p(b), _p(x), int(n_iter), int(bool(reorth)))
    return x


def _shape3(f, ndim):
    f = _c64(f)
    if f.ndim == 2:
        f = f[None]
    nz, ny, nx = f.shape
    assert ndim == 3 or nz == 1
    return f, nx, ny, nz


def face_mag2(f, ndim=2):
    f, nx, ny, nz = _shape3(f, ndim)
    out = np.zeros((ndim, nz, ny, nx))
    lib().orc_face_mag2(ndim, nx, ny, nz, _p(f), _p(out))
    return out


def sigma(n0sq, q, eps=1e-6):
    n0sq = _c64(n0sq)
    ndim, nz, ny, nx = n0sq.shape
    return float(lib().orc_sigma(ndim, nx, ny, nz, _p(n0sq), _f32(q), _f32(eps)))


def weights(n0sq, sig, mode=0):
    n0sq = _c64(n0sq)
    ndim, nz, ny, nx = n0sq.shape
    w = np.zeros_like(n0sq)
    lib().orc_weights(ndim, nx, ny, nz, _p(n0sq), float(sig), int(mode), _p(w))
    return w


def update_weights(f, q=0.90, eps=1e-6, mode=0, ndim=2):
    """O5 -> O6 -> O7.  Returns (w [ndim,nz,ny,nx], sigma)."""
    f, nx, ny, nz = _shape3(f, ndim)
    w = np.zeros((ndim, nz, ny, nx))
    s = lib().orc_update_weights(ndim, nx, ny, nz, _p(f), _f32(q), _f32(eps), int(mode), _p(w))
    return w, float(s)


def gradient(f, v, w, lam, eps=1e-6, ndim=2):
    f, nx, ny, nz = _shape3(f, ndim)
    v = _c64(v).reshape(f.shape)
    w = _c64(w).reshape((ndim,) + f.shape)
    g = np.zeros_like(f)
    lib().orc_gradient(ndim, nx, ny, nz, _p(f), _p(v), _p(w), _f32(lam), _f32(eps), _p(g))
    return g


def energy(f, v, w, lam, eps=1e-6, ndim=2):
    f, nx, ny, nz = _shape3(f, ndim)
    v = _c64(v).reshape(f.shape)
    w = _c64(w).reshape((ndim,) + f.shape)
    return float(lib().orc_energy(ndim, nx, ny, nz, _p(f), _p(v), _p(w), _f32(lam), _f32(eps)))


def eptv_step(f, v, w, lam, params=None, ndim=2):
    """One GD sweep (O8 + O9).  Returns (f_new, k, E0, G, t)."""
    f, nx, ny, nz = _shape3(f, ndim)
    f = f.copy()
    v = _c64(v).reshape(f.shape)
    w = _c64(w).reshape((ndim,) + f.shape)
    op = make_params(params or {})
    out = np.zeros(3)
    k = lib().orc_eptv_step(ndim, nx, ny, nz, _p(f), _p(v), _p(w), _f32(lam), C.byref(op), _p(out))
    return f, int(k), float(out[0]), float(out[1]), float(out[2])


def reconstruct(g, sino, params):
    """O10.  Returns (f [nz,ny,nx] or [ny,nx], w, log[n_outer*n_gd, 4] = (sigma,k,E0,G))."""
    og = make_geom(g)
    op = make_params(params)
    sino = _c64(sino)
    assert sino.size == og.nviews * og.nv * og.nu
    f = np.zeros((og.nz, og.ny, og.nx))
    w = np.zeros((og.ndim, og.nz, og.ny, og.nx))
    log = np.zeros((max(op.n_outer * op.n_gd, 1), 4))
    lib().orc_reconstruct(C.byref(og), _p(sino), C.byref(op), _p(f), _p(w), _p(log))
    if og.ndim == 2:
        return f[0], w[:, 0], log
    return f, w, log


# ---------------------------------------------------------------------------------------------
# NEXT rows of SURVEY.md 8(f), composed in numpy from the C steps above (no new arithmetic in C):
#   NEXT-1  CGLS with the paper's unmatched pair (P by ray tracing, P^T by Eq. (11))
#   NEXT-4  the plain gradient update (P1) of Eq. 8, that the paper replaced by CGLS
# Pins (tests/test_oracle_pins.py): cgls_recurrence(back_op=back) equals orc_cgls(reorth=0) - the C transcription
# of App. I, itself pinned to lstsq / hand iterations; p1_updates equals the dense-matrix iteration on 8x8 and
# converges to the least-squares solution; reconstruct_steps(step1 = cgls) equals orc_reconstruct bit for bit.
# ---------------------------------------------------------------------------------------------
def cgls_recurrence(g, b, x0, n_iter, back_op=None):
    """App. I as printed, with the backprojector given as a function (default: the exact
    transpose `back`; `back_eq11` gives the paper's own unmatched pair). Zero denominators stop (S4)."""
    back_op = back_op or back
    b = _c64(b)
    u = _c64(x0).copy()
    r = b - forward(g, u).reshape(b.shape)           # r = y - P u            (:420)
    gr = back_op(g, r).reshape(u.shape)              # g = P^T r
    s = gr.copy()
    gamma = float(np.sum(gr * gr))
    for _ in range(int(n_iter)):
        q = forward(g, s).reshape(b.shape)           # q = P s                (:423)
        delta = float(np.sum(q * q))
        if gamma == 0.0 or delta == 0.0:
            break
        a = gamma / delta
        u = u + a * s                                # :426
        r = r - a * q                                # :429
        gr = back_op(g, r).reshape(u.shape)
        gamma_new = float(np.sum(gr * gr))           # :432
        s = gr + (gamma_new / gamma) * s             # :435
        gamma = gamma_new
    return u


def p1_updates(g, y, f, n, tau, back_op=None):
    """(P1) of Eq. 8: f <- f - tau P^T (P f - y), n times; tau = mu/lambda."""
    back_op = back_op or back
    y = _c64(y)
    f = _c64(f).copy()
    tau = _f32(tau)
    for _ in range(int(n)):
        r = y - forward(g, f).reshape(y.shape)
        f = f + tau * back_op(g, r).reshape(f.shape)
    return f


def reconstruct_steps(g, sino, params, step1=None):
    """O10 composed from the oracle's steps, with Step 1 given as a function
    step1(f) -> v (default: CGLS with the config's n_cgls, reading S24). Returns (f, log[n_outer*n_gd, 4])."""
    og = make_geom(g)
    d = params.params_dict() if hasattr(params, "params_dict") else dict(params)
    p = make_params(d)
    if step1 is None:
        step1 = lambda f: cgls(g, sino, f, p.n_cgls).reshape(f.shape)  # noqa: E731
    f = np.zeros((og.nz, og.ny, og.nx))
    log = []
    for _ in range(p.n_outer):
        f = _c64(step1(f)).reshape(f.shape)                            # Step 1 (:171)
        v = f.copy()
        for _ in range(p.n_gd):                                        # Step 2 (:172)
            w, sig = update_weights(f, p.sigma_quantile, p.eps, p.weights_mode, ndim=og.ndim)
            f, k, e0, g2, _t = eptv_step(f, v, w, p.lam, d, ndim=og.ndim)
            log.append((sig, k, e0, g2))
        if p.positivity:                                               # Step 3 (:173)
            f = np.maximum(f, 0.0)
    return (f[0] if og.ndim == 2 else f), np.array(log)
