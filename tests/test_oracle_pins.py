"""Pins of the oracle (oracle/ctr_oracle.c) to things OTHER than itself: closed forms,
brute force written independently in numpy here, textbook/library routines, invariants
and a hand-evaluated example (tests/golden/a2_a3_4x4.json).  CPU only.
Citations: PAPER.md lines; O*/S* = readings in DESIGN.md."""
import json
import math
from pathlib import Path

import numpy as np
import pytest

from ctr_inputs import (Ellipse, analytic_sinogram, get_config, make_case, make_phantom,
                        rasterize, ray_endpoints, scaled_config)
from ctr_inputs.configs import Config

GOLD = Path(__file__).resolve().parent / "golden"


def tiny2d(**kw):
    base = dict(name="t2", index=90, ndim=2, nx=8, ny=8, nz=1, dx=1.5, dy=1.5, dz=1.0,
                nviews=12, nu=12, nv=1, du=2.0, dv=1.0, dso=541.0, dsd=949.0)
    base.update(kw)
    return Config(**base)


def tiny3d(**kw):
    base = dict(name="t3", index=91, ndim=3, nx=5, ny=4, nz=3, dx=1.5, dy=1.25, dz=2.0,
                nviews=7, nu=6, nv=5, du=2.5, dv=3.0, dso=100.0, dsd=160.0)
    base.update(kw)
    return Config(**base)


# ---------------------------------------------------------------- independent brute force
def box_chords(cfg, lo, hi):
    """Length of every source->bin segment inside the axis-aligned box [lo,hi] (slab clip)."""
    out = np.zeros((cfg.nviews, cfg.nv, cfg.nu))
    for k in range(cfg.nviews):
        S, D = ray_endpoints(cfg, k)
        d = D - S
        amin = np.zeros(d.shape[:-1])
        amax = np.ones(d.shape[:-1])
        for ax in range(3):
            with np.errstate(divide="ignore", invalid="ignore"):
                a1 = (lo[ax] - S[ax]) / d[..., ax]
                a2 = (hi[ax] - S[ax]) / d[..., ax]
            par = d[..., ax] == 0
            inside = (S[ax] >= lo[ax]) & (S[ax] < hi[ax])
            en = np.where(par, -np.inf if inside else np.inf, np.minimum(a1, a2))
            ex = np.where(par, np.inf if inside else -np.inf, np.maximum(a1, a2))
            amin = np.maximum(amin, en)
            amax = np.minimum(amax, ex)
        out[k] = np.maximum(amax - amin, 0.0) * np.linalg.norm(d, axis=-1)
    return out


def image_box(cfg):
    lo = np.array([cfg.cx - cfg.nx * cfg.dx / 2, cfg.cy - cfg.ny * cfg.dy / 2, cfg.cz - cfg.nz * cfg.dz / 2])
    hi = lo + np.array([cfg.nx * cfg.dx, cfg.ny * cfg.dy, cfg.nz * cfg.dz])
    return lo, hi


def brute_matrix(cfg):
    """Dense A[ray, voxel] = |ray ∩ voxel box| for every pair, no traversal."""
    lo, _ = image_box(cfg)
    A = np.zeros((cfg.nviews * cfg.nv * cfg.nu, cfg.nz * cfg.ny * cfg.nx))
    for k in range(cfg.nz):
        for j in range(cfg.ny):
            for i in range(cfg.nx):
                vlo = lo + np.array([i * cfg.dx, j * cfg.dy, k * cfg.dz])
                vhi = vlo + np.array([cfg.dx, cfg.dy, cfg.dz])
                A[:, (k * cfg.ny + j) * cfg.nx + i] = box_chords(cfg, vlo, vhi).ravel()
    return A


# ---------------------------------------------------------------- O1/O2: P
@pytest.mark.parametrize("name", ["c1", "c2"])
def test_forward_of_ones_is_box_chord(orc, name):
    """(i) P·1 = chord of each ray through the image box, closed form, to 1e-12."""
    cfg = get_config(name)
    got = orc.forward(cfg, np.ones((cfg.ny, cfg.nx)))
    want = box_chords(cfg, *image_box(cfg))[:, 0, :]
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(want)
    assert want.max() > 0


def test_forward_of_ones_3d(orc):
    cfg = tiny3d()
    got = orc.forward(cfg, np.ones((cfg.nz, cfg.ny, cfg.nx)))
    want = box_chords(cfg, *image_box(cfg))
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(want)


@pytest.mark.parametrize("cfg", [tiny2d(), tiny2d(nx=7, ny=5, dx=1.0, dy=2.0, cx=0.7, cy=-0.4, u_off=0.25),
                                 tiny2d(nviews=8, nu=11, theta0=0.0)],
                         ids=["8x8", "7x5-offcentre", "axis-parallel-central-ray"])
def test_dense_matrix_2d(orc, cfg):
    """(ii) every p_ij equals the brute-force ray∩pixel length; includes rays parallel to an
    axis through pixel interiors (odd nu: the central ray at theta = 0, 90, ...)."""
    A = orc.matrix(cfg)
    B = brute_matrix(cfg)
    assert A.shape == B.shape
    assert np.max(np.abs(A - B)) <= 1e-11
    assert (B > 0).sum() > 50


def test_dense_matrix_3d(orc):
    cfg = tiny3d()
    A = orc.matrix(cfg)
    B = brute_matrix(cfg)
    assert np.max(np.abs(A - B)) <= 1e-11
    rng = np.random.default_rng(3)
    x = rng.random((cfg.nz, cfg.ny, cfg.nx))
    y = rng.random((cfg.nviews, cfg.nv, cfg.nu))
    assert np.allclose(orc.forward(cfg, x).ravel(), B @ x.ravel(), rtol=0, atol=1e-11)
    assert np.allclose(orc.back(cfg, y).ravel(), B.T @ y.ravel(), rtol=0, atol=1e-11)


def test_forward_back_equal_dense_matrix_products(orc):
    cfg = tiny2d()
    B = brute_matrix(cfg)
    rng = np.random.default_rng(1)
    x = rng.standard_normal((cfg.ny, cfg.nx))
    y = rng.standard_normal((cfg.nviews, cfg.nu))
    assert np.allclose(orc.forward(cfg, x).ravel(), B @ x.ravel(), rtol=0, atol=1e-11)
    assert np.allclose(orc.back(cfg, y).ravel(), B.T @ y.ravel(), rtol=0, atol=1e-11)


def test_disk_chord_closed_form(orc):
    """(iii) uniform disk: P(raster) -> 2 rho sqrt(r^2 - d^2) with ~O(h) discretisation error."""
    errs = []
    for n, h in [(64, 1.5), (128, 0.75), (256, 0.375)]:
        cfg = scaled_config("c1", nx=n, ny=n, dx=h, dy=h)
        r, rho = 30.0, 0.02
        disk = [Ellipse(3.0, -2.0, 0, r, r, math.inf, 0.0, rho)]
        img = rasterize(cfg, disk, supersample=8)[0]
        got = orc.forward(cfg, img)
        # closed form written out here (not via ctr_inputs): distance of the disk centre to each ray
        want = np.zeros_like(got)
        for k in range(cfg.nviews):
            S, D = ray_endpoints(cfg, k)
            u = (D[0] - S)[:, :2]
            u /= np.linalg.norm(u, axis=1, keepdims=True)
            c = np.array([3.0, -2.0]) - S[:2]
            dist = np.abs(c[0] * u[:, 1] - c[1] * u[:, 0])
            want[k] = 2 * rho * np.sqrt(np.maximum(r * r - dist * dist, 0))
        errs.append(np.linalg.norm(got - want) / np.linalg.norm(want))
    assert errs[0] < 0.02
    assert errs[1] < 0.6 * errs[0] and errs[2] < 0.6 * errs[1]


@pytest.mark.parametrize("name,tol", [("c1", 0.03), ("c2", 0.008), ("c3", 0.005)])
def test_ellipse_phantom_analytic(orc, name, tol):
    """(iii) P(raster of the seeded phantom) vs analytic ellipse line integrals."""
    cfg = get_config(name)
    d = make_case(cfg, noisy=False)
    got = orc.forward(cfg, d["truth"][0].astype(np.float64))
    want = d["sino"][0].astype(np.float64)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < tol


def test_rotation_symmetry(orc):
    """(iv) rotating the image by 90 deg equals shifting the views by nviews/4."""
    cfg = scaled_config("c1", nviews=32)
    rng = np.random.default_rng(5)
    x = rng.random((cfg.ny, cfg.nx))
    s0 = orc.forward(cfg, x)
    # rotate the object by +90 deg: new[j][i] = old at (x,y) -> (y,-x)
    xr = np.rot90(x, k=1)  # counter-clockwise in (row=j=y up, col=i=x) with y increasing by row
    s1 = orc.forward(cfg, xr)
    a = np.linalg.norm(s1 - np.roll(s0, cfg.nviews // 4, axis=0))
    b = np.linalg.norm(s1 - np.roll(s0, -cfg.nviews // 4, axis=0))
    # dtheta is an fp32 value, so 8*dtheta misses pi/2 by ~1e-8 rad: tolerance 2e-6, not 1e-12
    assert min(a, b) <= 2e-6 * np.linalg.norm(s0)
    assert max(a, b) > 1e-3 * np.linalg.norm(s0)


def test_arc_detector_directions(orc):
    """ARC: bin a looks along angle theta + t_a/dsd at distance dsd."""
    cfg = tiny2d(det_type=1, nu=9, du=1.0239, dsd=949.075)
    for k in (0, 3, 7):
        th = cfg.theta0 + cfg.dtheta * k
        for a in (0, 4, 8):
            S, D = orc.ray(cfg, k, 0, a)
            d = D - S
            beta = (a - 4.0) * float(np.float32(1.0239)) / float(np.float32(949.075))
            assert abs(np.linalg.norm(d) - float(np.float32(949.075))) < 1e-9
            assert abs(math.atan2(d[1], d[0]) - math.atan2(math.sin(th + beta), math.cos(th + beta))) < 1e-12
    A = orc.matrix(cfg)
    B = brute_matrix(cfg)
    assert np.max(np.abs(A - B)) <= 1e-11


# ---------------------------------------------------------------- O3: P^T
@pytest.mark.parametrize("name", ["c1", "c2"])
def test_adjoint_identity(orc, name):
    """PAPER.md:471 (A3'): <f, P^T y> = <P f, y>; exact transpose -> 1e-12."""
    cfg = get_config(name)
    rng = np.random.default_rng(7)
    x = rng.standard_normal((cfg.ny, cfg.nx))
    y = rng.standard_normal((cfg.nviews, cfg.nu))
    px, pty = orc.forward(cfg, x), orc.back(cfg, y)
    assert abs((px * y).sum() - (x * pty).sum()) <= 1e-12 * np.linalg.norm(px) * np.linalg.norm(y)


# ---------------------------------------------------------------- O4: CGLS
def test_cgls_converges_to_dense_least_squares(orc):
    """CGLS from x0 = 0 -> the min-norm least-squares solution (textbook)."""
    cfg = tiny2d()
    A = brute_matrix(cfg)
    rng = np.random.default_rng(11)
    b = A @ rng.random(cfg.nx * cfg.ny) + 0.01 * rng.standard_normal(A.shape[0])
    x_ls = np.linalg.lstsq(A, b, rcond=None)[0]
    x = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), np.zeros((cfg.ny, cfg.nx)), 400, reorth=False).ravel()
    assert np.linalg.norm(A @ x - A @ x_ls) <= 1e-8 * np.linalg.norm(b)
    assert np.linalg.norm(x - x_ls) <= 1e-6 * np.linalg.norm(x_ls)
    # re-orthogonalised: finite termination after at most rank(A) = 64 steps
    x = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), np.zeros((cfg.ny, cfg.nx)), 64, reorth=True).ravel()
    assert np.linalg.norm(A @ x - A @ x_ls) <= 1e-8 * np.linalg.norm(b)


def test_cgls_first_iterate_and_monotone_residual(orc):
    cfg = tiny2d()
    A = brute_matrix(cfg)
    rng = np.random.default_rng(12)
    b = rng.random(A.shape[0])
    x0 = rng.random(A.shape[1])
    r0 = b - A @ x0
    s0 = A.T @ r0
    x1_hand = x0 + (s0 @ s0) / ((A @ s0) @ (A @ s0)) * s0            # App. I steps 1-2, m = 0
    x1 = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), x0.reshape(cfg.ny, cfg.nx), 1).ravel()
    assert np.allclose(x1, x1_hand, rtol=0, atol=1e-12)
    # two iterations against the recurrence typed from App. I (:423-435)
    a0 = (s0 @ s0) / ((A @ s0) @ (A @ s0))
    r1 = r0 - a0 * (A @ s0)
    g1 = A.T @ r1
    s1 = g1 + (g1 @ g1) / (s0 @ s0) * s0
    x2_hand = x1_hand + (g1 @ g1) / ((A @ s1) @ (A @ s1)) * s1
    x2 = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), x0.reshape(cfg.ny, cfg.nx), 2).ravel()
    assert np.allclose(x2, x2_hand, rtol=0, atol=1e-12)
    res = [np.linalg.norm(b - A @ orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu),
                                           x0.reshape(cfg.ny, cfg.nx), m).ravel()) for m in range(0, 12)]
    assert all(res[m + 1] <= res[m] * (1 + 1e-12) for m in range(11))
    # n_iter = 0 is the identity
    assert np.array_equal(orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), x0.reshape(cfg.ny, cfg.nx), 0).ravel(), x0)


def krylov_minimiser(A, b, x0, n):
    """The DEFINITION of the n-th CGLS iterate (Hestenes & Stiefel): argmin ||A x - b|| over
    x0 + span{(A^T A)^i A^T r0, i < n}. Built without any CG recurrence: an orthonormal Krylov
    basis by Arnoldi with doubly applied Gram-Schmidt in extended precision, then a small dense
    least-squares solve."""
    L = np.longdouble
    A_, r0 = A.astype(L), (b - A @ x0).astype(L)
    v = A_.T @ r0
    Q = []
    for i in range(n):
        for _ in range(2):
            for q in Q:
                v = v - (q @ v) * q
        nv = np.sqrt(v @ v)
        if nv == 0:
            break
        Q.append(v / nv)
        v = A_.T @ (A_ @ Q[-1])
    Qm = np.stack(Q, axis=1)
    AQ = (A_ @ Qm).astype(np.float64)
    c = np.linalg.lstsq(AQ, r0.astype(np.float64), rcond=None)[0]
    return x0 + Qm.astype(np.float64) @ c


@pytest.mark.parametrize("n", [1, 3, 6, 10, 15])
def test_cgls_iterate_is_the_krylov_subspace_minimiser(orc, n):
    """Pins the re-orthogonalised CGLS (reading S24) to the textbook definition of the iterate,
    and shows the recurrence as printed agrees with it while it is still numerically orthogonal."""
    cfg = tiny2d()
    A = brute_matrix(cfg)
    rng = np.random.default_rng(16)
    b = A @ rng.random(A.shape[1]) + 0.05 * rng.standard_normal(A.shape[0])
    x0 = 0.1 * rng.random(A.shape[1])
    want = krylov_minimiser(A, b, x0, n)
    got = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), x0.reshape(cfg.ny, cfg.nx), n, reorth=True).ravel()
    assert np.linalg.norm(got - want) <= 1e-9 * np.linalg.norm(want)
    plain = orc.cgls(cfg, b.reshape(cfg.nviews, cfg.nu), x0.reshape(cfg.ny, cfg.nx), n, reorth=False).ravel()
    if n <= 6:
        assert np.linalg.norm(plain - want) <= 1e-9 * np.linalg.norm(want)


def test_cgls_reorthogonalised_is_reproducible_where_the_printed_recurrence_is_not(orc):
    """Reading S24, measured on the seeded c1 workload with 15 iterations: a 1e-13 relative
    perturbation of y moves the printed recurrence's result by orders of magnitude more than the
    re-orthogonalised one (loss of orthogonality once the dominant singular direction converged)."""
    cfg = get_config("c1")
    y = make_case(cfg)["sino"][0].astype(np.float64)
    yp = y * (1 + 1e-13 * np.random.default_rng(17).standard_normal(y.shape))
    z = np.zeros((cfg.ny, cfg.nx))
    d = {}
    for re in (False, True):
        a, b = orc.cgls(cfg, y, z, 15, reorth=re), orc.cgls(cfg, yp, z, 15, reorth=re)
        d[re] = np.linalg.norm(a - b) / np.linalg.norm(a)
    assert d[True] <= 1e-10
    assert d[False] >= 1e3 * d[True]
    # early iterations: both variants are the same iterate
    a, b = orc.cgls(cfg, y, z, 5, reorth=False), orc.cgls(cfg, y, z, 5, reorth=True)
    assert np.linalg.norm(a - b) <= 1e-9 * np.linalg.norm(a)


# ---------------------------------------------------------------- O5-O8: A2 / A3
def test_hand_evaluated_4x4(orc):
    gold = json.loads((GOLD / "a2_a3_4x4.json").read_text())
    f = np.array(gold["image_rows_j_then_cols_i"], dtype=np.float64)
    n0 = orc.face_mag2(f)                                   # [axis, 0, j, i]
    for key, val in gold["n0sq"].items():
        ax, i, j = key.split("_")
        assert n0[0 if ax == "x" else 1, 0, int(j), int(i)] == pytest.approx(val, abs=1e-13)
    ones = (n0 > -1).astype(np.float64)
    g_tv = orc.gradient(f, f, orc.weights(n0, 1.0, mode=1), lam=0.0, eps=0.0)
    assert g_tv[0, 1, 1] == pytest.approx(gold["a2_tv_at_1_1"], abs=5e-8)
    w = orc.weights(n0, gold["sigma"], mode=0)
    for key, val in gold["omega"].items():
        ax, i, j = key.split("_")
        assert w[0 if ax == "x" else 1, 0, int(j), int(i)] == pytest.approx(val, abs=5e-9)
    g_ep = orc.gradient(f, f, w, lam=0.0, eps=0.0)
    assert g_ep[0, 1, 1] == pytest.approx(gold["a2_eptv_at_1_1"], abs=5e-8)
    assert ones.all()


def test_constant_image_invariants(orc):
    """north_star invariant: zero TV and unit weights on a constant image (S12)."""
    for shape, ndim in (((1, 9, 7), 2), ((4, 5, 6), 3)):
        f = np.full(shape, 0.37)
        n0 = orc.face_mag2(f, ndim)
        assert np.all(n0 == 0)
        w, sig = orc.update_weights(f, 0.9, 1e-6, 0, ndim)
        assert sig == pytest.approx(float(np.float32(1e-6)))
        interior = np.ones_like(w, dtype=bool)
        interior[0, :, :, -1] = False
        interior[1, :, -1, :] = False
        if ndim == 3:
            interior[2, -1, :, :] = False
        assert np.all(w[interior] == 1.0) and np.all(w[~interior] == 0.0)
        assert np.all(orc.gradient(f, f, w, 0.02, 1e-6, ndim) == 0)
        assert orc.energy(f, f, w, 0.02, 1e-6, ndim) == 0.0


def test_ramp_has_zero_interior_tv_gradient(orc):
    j, i = np.mgrid[0:10, 0:12]
    f = (0.3 * i - 0.2 * j + 1.0)[None]
    w = np.ones((2,) + f.shape)
    w[0, :, :, -1] = 0
    w[1, :, -1, :] = 0
    g = orc.gradient(f, f, w, 0.0, 0.0)
    assert np.max(np.abs(g[0, 2:-2, 2:-2])) < 1e-12
    # on a ramp every interior face magnitude is the Euclidean gradient norm (isotropy, S5)
    n0 = orc.face_mag2(f)
    assert np.allclose(n0[0, 0, 2:-2, 2:-2], 0.3 ** 2 + 0.2 ** 2)
    assert np.allclose(n0[1, 0, 2:-2, 2:-2], 0.3 ** 2 + 0.2 ** 2)


def test_one_dimensional_reduction_to_textbook_tv(orc):
    """With a single row the transverse terms of A3 vanish: N0 = |f_{i+1}-f_i|, J = sum|diff|
    and (omega = 1) A2 = -(sign(d_i) - sign(d_{i-1})): the textbook 1D TV subgradient."""
    rng = np.random.default_rng(2)
    f = rng.standard_normal((1, 1, 40))
    n0 = orc.face_mag2(f)
    assert np.allclose(n0[0, 0, 0, :-1], np.diff(f[0, 0]) ** 2, atol=1e-15)
    assert np.all(n0[1] == 0)
    w = orc.weights(n0, 1.0, mode=1)
    # energy: (1/ndim) * sum |d|   (O9, eps = 0)
    assert orc.energy(f, f, w, 0.0, 0.0) == pytest.approx(np.abs(np.diff(f[0, 0])).sum() / 2, rel=1e-14)
    sgn = np.sign(np.diff(f[0, 0]))
    want = -(np.concatenate([sgn, [0]]) - np.concatenate([[0], sgn]))
    assert np.allclose(orc.gradient(f, f, w, 0.0, 0.0)[0, 0], want, atol=1e-12)


def test_gradient_matches_energy_derivative_in_1d(orc):
    """In 1D A2 IS the derivative of the discrete energy (times ndim, as E carries 1/ndim):
    central differences of orc_energy pin the sign and indexing of A2 and of lambda(f-v)."""
    rng = np.random.default_rng(4)
    f = rng.standard_normal((1, 1, 16))
    v = rng.standard_normal((1, 1, 16))
    n0 = orc.face_mag2(f)
    w = orc.weights(n0, 1.3, mode=0)
    eps, lam = 0.05, 0.7
    g = orc.gradient(f, v, w, lam, eps)[0, 0]
    g_fid = np.float32(lam) * (f - v)[0, 0]
    h = 1e-6
    for i in range(16):
        e = np.zeros_like(f)
        e[0, 0, i] = h
        dE_tv = (orc.energy(f + e, v, w, 0.0, eps) - orc.energy(f - e, v, w, 0.0, eps)) / (2 * h)
        dE_fid = (orc.energy(f + e, v, 0 * w, lam, eps) - orc.energy(f - e, v, 0 * w, lam, eps)) / (2 * h)
        assert g[i] - g_fid[i] == pytest.approx(2 * dE_tv, abs=1e-6)
        assert g_fid[i] == pytest.approx(dE_fid, abs=1e-6)


def test_flip_and_transpose_equivariance(orc):
    rng = np.random.default_rng(6)
    f = rng.random((1, 9, 11))
    v = rng.random((1, 9, 11))
    w, sig = orc.update_weights(f, 0.9)
    g = orc.gradient(f, v, w, 0.3)
    # left-right flip
    wf, sf = orc.update_weights(f[:, :, ::-1], 0.9)
    assert sf == pytest.approx(sig, rel=1e-14)
    assert np.allclose(orc.gradient(f[:, :, ::-1], v[:, :, ::-1], wf, 0.3), g[:, :, ::-1], atol=1e-13)
    # transpose swaps the roles of the x- and y-face planes
    ft, vt = f.transpose(0, 2, 1), v.transpose(0, 2, 1)
    wt, st = orc.update_weights(ft, 0.9)
    assert st == pytest.approx(sig, rel=1e-14)
    assert np.allclose(wt[0], w[1].transpose(0, 2, 1), atol=1e-14)
    assert np.allclose(orc.gradient(ft, vt, wt, 0.3), g.transpose(0, 2, 1), atol=1e-13)


def test_tv_is_eptv_with_unit_weights_and_eptv_le_tv(orc):
    """TV = EPTV with w = 1, and w < 1 => ||f||_EPTV <= ||f||_TV."""
    rng = np.random.default_rng(8)
    f = rng.random((1, 12, 12))
    w_tv, _ = orc.update_weights(f, 0.9, mode=1)
    w_ep, sig = orc.update_weights(f, 0.9, mode=0)
    interior = np.ones_like(w_tv, dtype=bool)
    interior[0, :, :, -1] = False
    interior[1, :, -1, :] = False
    assert np.all(w_tv[interior] == 1.0)
    assert np.all((w_ep[interior] > 0) & (w_ep[interior] <= 1.0))
    assert orc.energy(f, f, w_ep, 0.0) <= orc.energy(f, f, w_tv, 0.0)
    n0 = orc.face_mag2(f)
    assert np.allclose(w_ep[interior], np.exp(-n0[interior] / sig ** 2), rtol=1e-14)


def test_face_mag2_3d_against_direct_numpy(orc):
    """3D generalisation (S22) of A3, written out with numpy edge padding."""
    rng = np.random.default_rng(9)
    f = rng.random((4, 5, 6))
    n0 = orc.face_mag2(f, 3)
    fp = np.pad(f, 1, mode="edge")
    # x-faces: m = mean of the two voxels along x; transverse axes y (axis 1) and z (axis 0)
    m = 0.5 * (fp[:, :, 1:] + fp[:, :, :-1])          # [nz+2, ny+2, nx+1], face i between i-1+1.. (padded)
    mx = m[:, :, 1:-1]                                 # faces between voxel i and i+1, i = 0..nx-2
    d = f[:, :, 1:] - f[:, :, :-1]
    want = d ** 2
    for axis in (0, 1):
        c = mx[1:-1, 1:-1]
        up = np.take(mx, range(2, mx.shape[axis]), axis=axis)
        dn = np.take(mx, range(0, mx.shape[axis] - 2), axis=axis)
        other = 1 - axis
        up = np.take(up, range(1, up.shape[other] - 1), axis=other)
        dn = np.take(dn, range(1, dn.shape[other] - 1), axis=other)
        want = want + 0.5 * (up - c) ** 2 + 0.5 * (c - dn) ** 2
    assert np.allclose(n0[0, :, :, :-1], want, atol=1e-14)
    assert np.all(n0[0, :, :, -1] == 0)


def test_hand_evaluated_3x3x3(orc):
    """3D A2/A3 (reading S22) on a 3x3x3 volume evaluated by hand: all three face axes, both faces of every
    axis at the centre voxel, one border-plane face, TV and EP-TV gradient at the interior voxel."""
    gold = json.loads((GOLD / "a2_a3_3x3x3.json").read_text())
    f = np.array(gold["volume_planes_k_then_rows_j_then_cols_i"], dtype=np.float64)   # [k, j, i]
    assert f[1, 1, 1] == 4 and f[1, 1, 0] == 1 and f[1, 1, 2] == 2 and f[1, 0, 1] == 7 and f[0, 1, 1] == 5
    axis = {"x": 0, "y": 1, "z": 2}
    n0 = orc.face_mag2(f, 3)                                 # [axis, k, j, i]
    for key, val in gold["n0sq"].items():
        ax, i, j, k = key.split("_")
        assert n0[axis[ax], int(k), int(j), int(i)] == pytest.approx(val, abs=1e-13), key
    g_tv = orc.gradient(f, f, orc.weights(n0, 1.0, mode=1), lam=0.0, eps=0.0, ndim=3)
    assert g_tv[1, 1, 1] == pytest.approx(gold["a2_tv_at_1_1_1"], abs=5e-8)
    w = orc.weights(n0, gold["sigma"], mode=0)
    for key, val in gold["omega"].items():
        ax, i, j, k = key.split("_")
        assert w[axis[ax], int(k), int(j), int(i)] == pytest.approx(val, abs=5e-9), key
    g_ep = orc.gradient(f, f, w, lam=0.0, eps=0.0, ndim=3)
    assert g_ep[1, 1, 1] == pytest.approx(gold["a2_eptv_at_1_1_1"], abs=5e-8)


def _face_mag2_numpy(f, A):
    """N0^2 of the +A faces of a volume f[k, j, i] written out directly from A3 with numpy
    edge padding (S12); numpy axis of image axis A (0 = x, 1 = y, 2 = z) is 2 - A. Border faces excluded."""
    na = 2 - A
    fp = np.pad(f, 1, mode="edge")
    lo = np.take(fp, range(0, fp.shape[na] - 1), axis=na)
    hi = np.take(fp, range(1, fp.shape[na]), axis=na)
    m = 0.5 * (hi + lo)                                      # face means, padded transversally
    d = hi - lo
    inner = [slice(1, -1)] * 3
    inner[na] = slice(1, -1)                                 # faces between voxel p and p+1, p = 0..n-2
    want = d[tuple(inner)] ** 2
    c = m[tuple(inner)]
    for T in range(3):
        if T == A:
            continue
        nt = 2 - T
        up, dn = list(inner), list(inner)
        up[nt], dn[nt] = slice(2, None), slice(0, -2)
        want = want + 0.5 * (m[tuple(up)] - c) ** 2 + 0.5 * (c - m[tuple(dn)]) ** 2
    return want


@pytest.mark.parametrize("A", [0, 1, 2])
def test_face_mag2_3d_every_axis_against_direct_numpy(orc, A):
    """x-, y- AND z-faces of the 3D A3 (S22): a wrong transverse axis or stride on any face axis fails here."""
    rng = np.random.default_rng(19 + A)
    f = rng.random((4, 5, 6))                                # [nz, ny, nx], all different
    n0 = orc.face_mag2(f, 3)
    want = _face_mag2_numpy(f, A)
    sl = [slice(None)] * 3
    sl[2 - A] = slice(0, -1)
    assert np.allclose(n0[A][tuple(sl)], want, atol=1e-14)
    sl[2 - A] = -1
    assert np.all(n0[A][tuple(sl)] == 0)
    # and the 2D routine is the 3D one on a single plane (no z terms)
    n2 = orc.face_mag2(f[:1], 2)
    assert np.allclose(n2[0, 0, :, :-1], _face_mag2_2d(f[0], 0), atol=1e-14)
    assert np.allclose(n2[1, 0, :-1, :], _face_mag2_2d(f[0], 1), atol=1e-14)


def _face_mag2_2d(f, A):
    fp = np.pad(f, 1, mode="edge")
    if A == 1:
        return _face_mag2_2d(f.T, 0).T
    m = 0.5 * (fp[:, 1:] + fp[:, :-1])[:, 1:-1]
    d = f[:, 1:] - f[:, :-1]
    return d ** 2 + 0.5 * (m[2:] - m[1:-1]) ** 2 + 0.5 * (m[1:-1] - m[:-2]) ** 2


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_gradient_matches_energy_derivative_on_3d_columns(orc, axis):
    """A column along one axis of a 3D volume: the transverse terms of A3 vanish (clamped indices), so A2 is
    the derivative of the discrete energy times ndim = 3 (E carries 1/ndim, O9/S22). Pins the stride of every
    axis, the sign of the flux difference and the 1/ndim factor at 3."""
    rng = np.random.default_rng(24 + axis)
    n = 9
    shape = [1, 1, 1]
    shape[axis] = n                                          # numpy axes [k, j, i]
    f, v = rng.standard_normal(shape), rng.standard_normal(shape)
    A = 2 - axis                                             # image axis of the column
    n0 = orc.face_mag2(f, 3)
    assert np.allclose(np.delete(n0, A, axis=0), 0.0)
    assert np.allclose(n0[A].ravel()[:-1], np.diff(f.ravel()) ** 2, atol=1e-15)
    w = orc.weights(n0, 1.3, mode=0)
    eps, lam = 0.05, 0.7
    g = orc.gradient(f, v, w, lam, eps, ndim=3).ravel()
    g_fid = np.float32(lam) * (f - v).ravel()
    h = 1e-6
    for i in range(n):
        e = np.zeros(n)
        e[i] = h
        e = e.reshape(shape)
        dE_tv = (orc.energy(f + e, v, w, 0.0, eps, ndim=3) - orc.energy(f - e, v, w, 0.0, eps, ndim=3)) / (2 * h)
        dE_fid = (orc.energy(f + e, v, 0 * w, lam, eps, ndim=3) - orc.energy(f - e, v, 0 * w, lam, eps, ndim=3)) / (2 * h)
        assert g[i] - g_fid[i] == pytest.approx(3 * dE_tv, abs=1e-6)
        assert g_fid[i] == pytest.approx(dE_fid, abs=1e-6)


def test_axis_permutation_equivariance_3d(orc):
    """Permuting the axes of the volume permutes the face planes and the gradient accordingly (S8/S22)."""
    rng = np.random.default_rng(27)
    f, v = rng.random((4, 5, 6)), rng.random((4, 5, 6))
    w, sig = orc.update_weights(f, 0.9, 1e-4, 0, ndim=3)
    g = orc.gradient(f, v, w, 0.3, 1e-4, ndim=3)
    e0 = orc.energy(f, v, w, 0.3, 1e-4, ndim=3)
    for perm in ((0, 2, 1), (2, 1, 0), (1, 0, 2), (1, 2, 0)):      # numpy axes [k, j, i] -> permuted
        fp, vp = np.ascontiguousarray(f.transpose(perm)), np.ascontiguousarray(v.transpose(perm))
        wp, sp = orc.update_weights(fp, 0.9, 1e-4, 0, ndim=3)
        assert sp == pytest.approx(sig, rel=1e-14)
        for A in range(3):
            # image axis A of the permuted volume is numpy axis 2 - A, which was numpy axis perm[2 - A]
            assert np.allclose(wp[A], w[2 - perm[2 - A]].transpose(perm), atol=1e-14)
        assert np.allclose(orc.gradient(fp, vp, wp, 0.3, 1e-4, ndim=3), g.transpose(perm), atol=1e-13)
        assert orc.energy(fp, vp, wp, 0.3, 1e-4, ndim=3) == pytest.approx(e0, rel=1e-13)


# ---------------------------------------------------------------- O6: sigma
@pytest.mark.parametrize("q", [0.5, 0.9, 0.95, 1.0, 1e-9])
def test_sigma_is_order_statistic(orc, q):
    rng = np.random.default_rng(10)
    f = rng.random((1, 13, 17))
    n0 = orc.face_mag2(f)
    S = np.sqrt(np.concatenate([n0[0, 0, :, :-1].ravel(), n0[1, 0, :-1, :].ravel()]))
    assert len(S) == 12 * 17 + 13 * 16
    k = min(max(math.ceil(float(np.float32(q)) * len(S)), 1), len(S))
    assert orc.sigma(n0, q, 1e-6) == np.sort(S)[k - 1]
    assert orc.sigma(n0, q, 10.0) == 10.0  # floor at eps


# ---------------------------------------------------------------- O9: Armijo sweep
def test_armijo_accepts_first_sufficient_decrease(orc):
    rng = np.random.default_rng(13)
    v = 0.02 + 0.004 * rng.standard_normal((1, 24, 24))
    f = v.copy()
    p = dict(armijo_t0=1e-3, armijo_rho=0.5, armijo_c=1e-4, armijo_max=16, eps=1e-6)
    lam = 0.02
    E_prev = None
    ks = []
    for sweep in range(6):
        w, sig = orc.update_weights(f, 0.9)
        g = orc.gradient(f, v, w, lam)
        f_new, k, E0, G, t = orc.eptv_step(f, v, w, lam, p)
        assert G == pytest.approx((g ** 2).sum(), rel=1e-13)
        assert E0 == pytest.approx(orc.energy(f, v, w, lam), rel=1e-13)
        assert k >= 0
        t0, rho, c = (float(np.float32(p[x])) for x in ("armijo_t0", "armijo_rho", "armijo_c"))
        assert t == pytest.approx(t0 * rho ** k)
        assert np.allclose(f_new, f - t * g, atol=1e-18)
        E1 = orc.energy(f_new, v, w, lam)
        assert E1 <= E0 - c * t * G                                   # the inequality holds at t
        for kk in range(k):                                           # and fails at every larger t
            tt = t0 * rho ** kk
            assert orc.energy(f - tt * g, v, w, lam) > E0 - c * tt * G
        assert E1 <= E0                                               # monotone within the sweep (S17)
        ks.append(k)
        f = f_new


def test_armijo_rejects_everything_leaves_f_unchanged(orc):
    rng = np.random.default_rng(14)
    v = rng.random((1, 10, 10))
    f = v + 0.1 * rng.standard_normal(v.shape)
    w, _ = orc.update_weights(f, 0.9)
    # a huge first step and only one trial: cannot decrease the energy
    f_new, k, E0, G, t = orc.eptv_step(f, v, w, 0.02, dict(armijo_t0=1e3, armijo_max=1))
    assert k == -1 and t == 0.0
    assert np.array_equal(f_new, f)


# ---------------------------------------------------------------- O10: outer loop
def test_reconstruct_positivity_and_restarted_cgls(orc):
    cfg = tiny2d()
    A = brute_matrix(cfg)
    rng = np.random.default_rng(15)
    x_true = rng.random(cfg.nx * cfg.ny)
    b = (A @ x_true).reshape(cfg.nviews, cfg.nu)
    # n_gd = 0, no clamp: the outer loop is restarted CGLS (S1): identical to chaining orc.cgls,
    # and it drives the (consistent) system's residual towards the dense least-squares one (= 0)
    f, w, log = orc.reconstruct(cfg, b, dict(n_outer=30, n_cgls=20, n_gd=0, positivity=0))
    u = np.zeros((cfg.ny, cfg.nx))
    res = []
    for it in range(30):
        u = orc.cgls(cfg, b, u, 20)
        res.append(np.linalg.norm(A @ u.ravel() - b.ravel()))
    assert np.array_equal(f, u)
    x_ls = np.linalg.lstsq(A, b.ravel(), rcond=None)[0]
    assert np.linalg.norm(A @ x_ls - b.ravel()) <= 1e-9 * np.linalg.norm(b)
    assert all(res[i + 1] <= res[i] for i in range(29))
    assert res[-1] <= 5e-4 * np.linalg.norm(b)
    # one outer iteration by composition of the pinned parts
    p = dict(n_outer=1, n_cgls=4, n_gd=3, lam=0.05, positivity=1)
    f1, w1, log1 = orc.reconstruct(cfg, b - 0.3, p)
    u = orc.cgls(cfg, b - 0.3, np.zeros((cfg.ny, cfg.nx)), 4)
    fm = u.copy()
    for s in range(3):
        ww, sig = orc.update_weights(fm, 0.9)
        fm3, k, E0, G, t = orc.eptv_step(fm, u, ww, 0.05, p)
        assert log1[s, 0] == sig and log1[s, 1] == k and log1[s, 2] == E0
        fm = fm3[0]
    assert np.array_equal(f1, np.maximum(fm, 0.0))
    assert f1.min() >= 0.0 and (fm < 0).any()
    assert np.array_equal(w1, ww[:, 0])


def test_composed_outer_loop_is_orc_reconstruct(orc):
    """tests/golden/make_c5_golden.py composes O10 from the oracle's own steps so that it can checkpoint a long
    run: the composition must be orc_reconstruct itself, bit for bit (2D and 3D)."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_c5_golden", GOLD / "make_c5_golden.py")
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    cfg2 = scaled_config("c1", n_outer=2, n_cgls=4, n_gd=3)
    cfg3 = tiny3d(nx=10, ny=9, nz=6, nviews=8, nu=14, nv=10, n_outer=2, n_cgls=3, n_gd=2, lam=0.02)
    rng = np.random.default_rng(12)
    for cfg, sino in ((cfg2, make_case(cfg2)["sino"][0].astype(np.float64)),
                      (cfg3, rng.random((cfg3.nviews, cfg3.nv, cfg3.nu)))):
        want, _, log = orc.reconstruct(cfg, sino, cfg)
        seen = []
        got, glog = mod.composed_reconstruct(orc, cfg, sino, cfg.n_outer, lambda n, f, lg: seen.append(n))
        assert np.array_equal(got.reshape(want.shape), want)
        assert np.array_equal(glog[:, 1], log[:, 1])                       # Armijo indices
        assert np.allclose(glog, log, rtol=1e-12, atol=0)                  # E0 is an OpenMP reduction: order may differ
        assert seen == [1, 2]


def test_reconstruct_c1_reduces_error_and_stays_positive(orc):
    """Sanity on the seeded c1 workload: positivity after every outer iteration
    and a reconstruction closer to the truth than the zero image."""
    cfg = scaled_config("c1", n_outer=3)
    d = make_case(cfg)
    f, w, log = orc.reconstruct(cfg, d["sino"][0], cfg)
    truth = d["truth"][0]
    assert f.min() >= 0.0
    assert np.linalg.norm(f - truth) < 0.5 * np.linalg.norm(truth)
    assert np.all(log[:, 1] >= 0)


# ------------------------------------------------------------------ S25: the composed iteration is well posed
def test_reconstruct_is_reproducible_under_the_S25_constants(orc):
    """DESIGN.md S25. With Armijo c = 1e-4 and eps = 1e-6 (a legal reading of PAPER.md:149, which gives no
    constants) the composed iteration amplifies a 1e-8 relative perturbation of the sinogram by > 1e4 on
    configs[0] (overshooting steps on a nearly non-smooth term: no fp32 implementation can track it to
    north_star's 1e-3). With c = 1/2 (never beyond the line minimiser of a quadratic) and eps = 1e-4 the
    amplification is that of the restarted CGLS alone (< 50)."""
    from ctr_inputs import make_case, scaled_config
    rng = np.random.default_rng(5)

    def amplification(cfg, p=1e-8):
        y = make_case(cfg, raster=False)["sino"][0].astype(np.float64)
        base, _, _ = orc.reconstruct(cfg, y, cfg)
        pert, _, _ = orc.reconstruct(cfg, y * (1 + p * rng.standard_normal(y.shape)), cfg)
        return np.linalg.norm(pert - base) / np.linalg.norm(base) / p

    cfg = scaled_config("c1")
    assert (float(np.float32(cfg.armijo_c)), float(np.float32(cfg.eps))) == (0.5, float(np.float32(1e-4)))
    assert amplification(cfg) < 50
    assert amplification(scaled_config("c1", n_gd=0)) < 50          # restarted CGLS alone
    assert amplification(scaled_config("c1", armijo_c=1e-4, eps=1e-6)) > 1e3


def test_S25_amplification_on_c2(orc):
    """DESIGN.md S25 on configs[1] at its full schedule (20 x (10 CGLS + 5 GD)): the constants first proposed
    (Armijo c = 1e-4, eps = 1e-6) amplify a 1e-8 perturbation of the data by > 1e3 (DESIGN.md quotes 2e5), the
    built ones (c = 1/2, eps = 1e-4) by < 100 (quoted: 22)."""
    rng = np.random.default_rng(5)
    cfg = get_config("c2")
    y = make_case(cfg, raster=False)["sino"][0].astype(np.float64)
    yp = y * (1 + 1e-8 * rng.standard_normal(y.shape))

    def amplification(c):
        base, _, _ = orc.reconstruct(c, y, c)
        pert, _, _ = orc.reconstruct(c, yp, c)
        return np.linalg.norm(pert - base) / np.linalg.norm(base) / 1e-8

    built = amplification(cfg)
    proposed = amplification(scaled_config("c2", armijo_c=1e-4, eps=1e-6))
    print(f"[S25] c2 amplification of a 1e-8 perturbation: built constants {built:.1f}, first proposal {proposed:.3g}")
    assert built < 100
    assert proposed > 1e3


def _cgls_fp32_emulation(orc, cfg, y, M, select):
    """The CUDA path's arithmetic emulated with the oracle's operators: fp64 recurrence, but P, P^T and every
    stored vector rounded to fp32; each new gradient is projected against the unit gradients select(n) picks out
    of the n stored so far (App. I; S24)."""
    f32 = lambda a: a.astype(np.float32).astype(np.float64)
    P = lambda x: f32(orc.forward(cfg, x))
    PT = lambda r: f32(orc.back(cfg, r))
    u = np.zeros((cfg.ny, cfg.nx))
    r = y.copy()
    g = PT(r)
    gam = (g * g).sum()
    s = g.copy()
    B = [g / np.sqrt(gam)]
    for _ in range(M):
        q = P(s)
        a = gam / (q * q).sum()
        u = f32(u + a * s)
        r = f32(r - a * q)
        g = PT(r)
        for i in select(len(B)):
            g = g - (B[i] * g).sum() * B[i]
        g = f32(g)
        gn = (g * g).sum()
        s = f32(g + gn / gam * s)
        gam = gn
        B.append(g / np.sqrt(gn))
    return u


@pytest.mark.parametrize("name", ["c1", "c2"])
def test_S24_projecting_against_the_first_four_gradients_tracks_the_full_reorthogonalisation(orc, name):
    """DESIGN.md S24, table rows "nothing", "first 4", "all": in fp32-rounded arithmetic the printed recurrence
    drifts from the exact-arithmetic iterate (the oracle's fully re-orthogonalised CGLS) by ~1e-2 after 10
    iterations, while projecting each new gradient against the FIRST FOUR unit gradients only - what the CUDA
    path does (CTR_MAX_BASIS = 4) - stays as close to it as projecting against all of them."""
    cfg = scaled_config(name, batch=1)
    y = make_case(cfg, raster=False)["sino"][0].astype(np.float64)
    M = 10
    ref = orc.cgls(cfg, y, np.zeros((cfg.ny, cfg.nx)), M)
    rel = lambda a: np.linalg.norm(a - ref) / np.linalg.norm(ref)
    none = rel(_cgls_fp32_emulation(orc, cfg, y, M, lambda n: []))
    first4 = rel(_cgls_fp32_emulation(orc, cfg, y, M, lambda n: range(min(4, n))))
    full = rel(_cgls_fp32_emulation(orc, cfg, y, M, lambda n: range(n)))
    print(f"[S24] {name}, {M} iterations, fp32-rounded emulation vs the oracle: nothing {none:.2e}, first 4 {first4:.2e}, all {full:.2e}")
    assert none >= 3e-3
    assert first4 <= 5e-5 and full <= 5e-5
    assert first4 <= 3 * full + 1e-6


def _cgls_fp32_lazy_emulation(orc, cfg, y, M, NB=4):
    """The CUDA path's LAZY phase (ctr_api.cu, S24) emulated the same way: the first NB iterations project
    in image space as above; from then on the coefficients c_i = <P b_i, r> are taken on the sinogram side, with
    P b_i = (q_i - beta_i q_(i-1)) / ||g'_i|| from the q = P s of the first iterations, the direction is carried as
    s_hat = g + beta s_hat with s = s_hat - sum e_i b_i, e_i <- c_i + beta e_i, q = P s_hat - sum e_i P b_i, and
    u = u_hat - sum d_i b_i (d_i += a e_i) is formed once at the end. Scalars are rounded to fp32 as on the device."""
    f32 = lambda a: np.asarray(a).astype(np.float32).astype(np.float64)
    P = lambda x: f32(orc.forward(cfg, x))
    PT = lambda r: f32(orc.back(cfg, r))
    u = np.zeros((cfg.ny, cfg.nx))
    r = y.copy()
    g = PT(r)
    gam = (g * g).sum()
    s = g.copy()
    ginv = 1.0 / np.sqrt(gam)
    B, PB = [f32(g * ginv)], []
    e, dacc = np.zeros(NB), np.zeros(NB)
    qprev, beta = None, 0.0
    for m in range(M):
        q = P(s)
        if m < NB:
            PB.append(f32(q * ginv if m == 0 else (q - beta * qprev) * ginv))
            qprev = q
        else:
            q = f32(q - sum(ei * pb for ei, pb in zip(e, PB)))
        a = float(np.float32(gam / (q * q).sum()))
        u = f32(u + a * s)
        dacc = dacc + a * e
        r = f32(r - a * q)
        g = PT(r)
        g2 = (g * g).sum()
        if m + 1 < NB:
            c = [float(np.float32((b * g).sum())) for b in B]
            g2 -= sum(ci * ci for ci in c)
            gp = g - sum(ci * b for ci, b in zip(c, B))
            beta = float(np.float32(g2 / gam))
            s = f32(gp + beta * s)
            ginv = 1.0 / np.sqrt(g2)
            B.append(f32(gp * ginv))
        else:
            c = np.array([float(np.float32((pb * r).sum())) for pb in PB])
            g2 -= (c * c).sum()
            beta = float(np.float32(g2 / gam))
            e = f32(c + beta * e)
            s = f32(g + beta * s)
        gam = g2
    return f32(u - sum(di * b for di, b in zip(dacc, B)))


@pytest.mark.parametrize("name,M", [("c1", 10), ("c2", 15)])
def test_S24_sinogram_side_projection_tracks_the_full_reorthogonalisation(orc, name, M):
    """DESIGN.md S24, lazy phase: moving the projection against the first four unit gradients to the sinogram side
    (<b_i, P^T r> = <P b_i, r>) and carrying the projected direction implicitly is the same iteration in exact
    arithmetic; in fp32-rounded arithmetic it stays as close to the oracle's fully re-orthogonalised CGLS as the
    image-space projection does."""
    cfg = scaled_config(name, batch=1)
    y = make_case(cfg, raster=False)["sino"][0].astype(np.float64)
    ref = orc.cgls(cfg, y, np.zeros((cfg.ny, cfg.nx)), M)
    rel = lambda a: np.linalg.norm(a - ref) / np.linalg.norm(ref)
    first4 = rel(_cgls_fp32_emulation(orc, cfg, y, M, lambda n: range(min(4, n))))
    lazy = rel(_cgls_fp32_lazy_emulation(orc, cfg, y, M))
    print(f"[S24] {name}, {M} iterations, fp32-rounded emulation vs the oracle: first 4 in image space {first4:.2e}, "
          f"lazy (sinogram side) {lazy:.2e}")
    assert lazy <= 5e-5
    assert lazy <= 3 * first4 + 1e-6


# ------------------------------------------------------------------ NEXT-1: the paper's backprojector Eq. (11)
def _paper_geometry(**kw):
    """arc detector, 888 units x 1.0239 mm, source-detector 949.075 mm, source-axis 541.0 mm;
    512 x 512 image over the 500 mm field of view (pixel size is not printed)."""
    from ctr_inputs.configs import Config
    base = dict(name="paper", index=91, ndim=2, nx=512, ny=512, nz=1, dx=500.0 / 512, dy=500.0 / 512, dz=1.0,
                nviews=40, nu=888, nv=1, du=1.0239, dv=1.0, dso=541.0, dsd=949.075, det_type=1)
    base.update(kw)
    return Config(**base)


def _smooth_pair(cfg, seed=7):
    """Smooth image supported well inside the field of view and a smooth sinogram."""
    rng = np.random.default_rng(seed)
    jj, ii = np.mgrid[0:cfg.ny, 0:cfg.nx]
    x = (ii - cfg.nx / 2 + 0.5) * cfg.dx
    y = (jj - cfg.ny / 2 + 0.5) * cfg.dy
    f = np.zeros((cfg.ny, cfg.nx))
    R = 0.3 * cfg.nx * cfg.dx
    for _ in range(5):
        cx, cy = rng.uniform(-0.4 * R, 0.4 * R, 2)
        s = rng.uniform(0.15 * R, 0.3 * R)
        f += rng.uniform(0.5, 1.0) * np.exp(-((x - cx) ** 2 + (y - cy) ** 2) / (2 * s * s))
    kk, bb = np.mgrid[0:cfg.nviews, 0:cfg.nu]
    g = 1.0 + 0.5 * np.cos(2 * np.pi * kk / cfg.nviews + 0.3) * np.cos(3.0 * (bb / cfg.nu - 0.5)) \
        + 0.3 * np.sin(5.0 * (bb / cfg.nu - 0.5))
    return f, g


def test_eq11_adjoint_mismatch_below_one_percent_as_the_paper_reports(orc):
    """"Numerical experiments indicate that this condition [<f,P^T y> = <Pf,y>, A3'] is
    satisfied with numerical error less than 1%" - the one number the paper prints for an operator. Checked on
    the paper's scanner geometry with smooth f and y, P being the (pinned) Siddon projector."""
    cfg = _paper_geometry()
    f, y = _smooth_pair(cfg)
    lhs = float((f * orc.back_eq11(cfg, y)).sum())
    rhs = float((orc.forward(cfg, f) * y).sum())
    assert abs(lhs - rhs) <= 0.01 * abs(rhs)
    assert abs(lhs - rhs) > 1e-9 * abs(rhs)       # and it is NOT the exact transpose


@pytest.mark.parametrize("det_type", [1, 0])
def test_eq11_tends_to_the_exact_transpose_for_smooth_data(orc, det_type):
    """Eq. (11) discretises the continuous adjoint (App. III A7); so does the exact transpose of the Siddon
    matrix (pinned above). Pixel by pixel the two differ by a few per cent (the box footprint of a ray beats
    against the pixel grid), but their averages over fixed 32 mm blocks inside the field of view must agree,
    the better the finer the grids - for the paper's arc detector and for the flat-detector change of variable."""
    errs = []
    for n, nu in ((64, 96), (128, 192)):
        cfg = _paper_geometry(nx=n, ny=n, dx=256.0 / n, dy=256.0 / n, nu=nu, du=1.0239 * 888 / nu * 0.62,
                              nviews=24, det_type=det_type)
        _, y = _smooth_pair(cfg)
        B, m = n // 8, 8
        blk = lambda z: z.reshape(m, B, m, B).mean(axis=(1, 3))
        a, b = blk(orc.back_eq11(cfg, y)), blk(orc.back(cfg, y))
        jj, ii = np.mgrid[0:m, 0:m]
        inside = (ii - m / 2 + 0.5) ** 2 + (jj - m / 2 + 0.5) ** 2 < (0.35 * m) ** 2
        errs.append(np.linalg.norm((a - b)[inside]) / np.linalg.norm(b[inside]))
    assert errs[0] < 5e-3 and errs[1] < errs[0] / 3


def test_eq11_pixels_outside_the_fan_get_nothing(orc):
    cfg = _paper_geometry(nx=64, ny=64, dx=4.0, dy=4.0, nu=16, du=2.0, nviews=1)
    img = orc.back_eq11(cfg, np.ones((1, cfg.nu)))
    # view 0: source on the -x axis, central ray along +x; the 16-unit fan covers |y| < ~9 mm at the isocentre
    assert img[32, 32] > 0 and img[0, 32] == 0 and img[63, 32] == 0
    assert np.all(img >= 0)


# ------------------------------------------------------------------ NEXT-1 / NEXT-4 compositions (oracle/ctr_oracle.py)
def test_cgls_recurrence_in_numpy_is_the_printed_recurrence_of_the_c_oracle(orc):
    """cgls_recurrence() is App. I typed a second time, in numpy, with the backprojector as a
    parameter; with the exact transpose it must reproduce orc_cgls(reorth=0) - the C transcription that the lstsq,
    hand-iteration and Krylov pins above hold in place."""
    cfg = scaled_config("c1")
    d = make_case(cfg)
    y = d["sino"][0].astype(np.float64)
    rng = np.random.default_rng(3)
    for x0 in (np.zeros((cfg.ny, cfg.nx)), 0.01 * rng.random((cfg.ny, cfg.nx))):
        for n in (1, 4):
            want = orc.cgls(cfg, y, x0, n, reorth=False)
            got = orc.cgls_recurrence(cfg, y, x0, n)
            assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(want)


def test_cgls_with_the_unmatched_pair_still_reduces_the_residual(orc):
    """NEXT-1: the paper runs CGLS with P by ray tracing and P^T by Eq. (11). On its scanner
    geometry (arc detector) the unmatched pair must behave like the matched one over the first iterations - the
    residual ||P u - y|| falls, and stays within a few per cent of the matched pair's - which is the paper's
    argument for accepting a < 1 % adjoint mismatch."""
    cfg = _paper_geometry(nx=128, ny=128, dx=500.0 / 128, dy=500.0 / 128, nu=222, du=1.0239 * 4, nviews=30)
    f, _ = _smooth_pair(cfg)
    y = orc.forward(cfg, f)
    x0 = np.zeros_like(f)
    res = {}
    for name, op in (("matched", orc.back), ("eq11", orc.back_eq11)):
        res[name] = [np.linalg.norm(orc.forward(cfg, orc.cgls_recurrence(cfg, y, x0, n, back_op=op)) - y) for n in (1, 3, 6)]
    r0 = np.linalg.norm(y)
    assert res["eq11"][0] < 0.6 * r0 and res["eq11"][2] < res["eq11"][1] < res["eq11"][0]
    for a, b in zip(res["matched"], res["eq11"]):
        assert b <= 1.5 * a + 1e-3 * r0


def test_p1_updates_equal_the_dense_matrix_iteration_and_its_svd_closed_form(orc):
    """(P1) of Eq. 8: v = f - tau P^T (P f - y). On 8x8 with the brute-force dense matrix the
    n-step result is the Landweber iterate written with that matrix, and from f = 0 it has the textbook closed form
    in the SVD A = U S V^T:  f_n = sum_i (1 - (1 - tau s_i^2)^n) / s_i (u_i . y) v_i, which tends to the minimum-norm
    least-squares solution for tau < 2/||A||^2 (the residual falls monotonically on the way)."""
    cfg = tiny2d()
    A = brute_matrix(cfg)
    rng = np.random.default_rng(5)
    y = A @ rng.random(A.shape[1]) + 0.01 * rng.standard_normal(A.shape[0])
    tau = float(np.float32(1.0 / np.linalg.norm(A, 2) ** 2))
    f = rng.random(A.shape[1])
    want = f.copy()
    for _ in range(7):
        want = want - tau * (A.T @ (A @ want - y))
    got = orc.p1_updates(cfg, y.reshape(cfg.nviews, cfg.nu), f.reshape(cfg.ny, cfg.nx), 7, tau)
    assert np.linalg.norm(got.ravel() - want) <= 1e-12 * np.linalg.norm(want)
    U, S, Vt = np.linalg.svd(A, full_matrices=False)
    keep = S > 1e-10 * S[0]
    res = []
    for n in (1, 20, 150):
        fn = orc.p1_updates(cfg, y.reshape(cfg.nviews, cfg.nu), np.zeros((cfg.ny, cfg.nx)), n, tau).ravel()
        closed = Vt[keep].T @ ((1.0 - (1.0 - tau * S[keep] ** 2) ** n) / S[keep] * (U[:, keep].T @ y))
        assert np.linalg.norm(fn - closed) <= 1e-10 * np.linalg.norm(closed)
        res.append(np.linalg.norm(A @ fn - y))
    assert res[2] < res[1] < res[0] < np.linalg.norm(y)


def test_reconstruct_steps_with_cgls_is_orc_reconstruct(orc):
    """reconstruct_steps() composes O10 with Step 1 as a parameter; with the default Step 1 it is orc_reconstruct."""
    cfg = scaled_config("c1", n_outer=2, n_cgls=4, n_gd=3)
    sino = make_case(cfg)["sino"][0].astype(np.float64)
    want, _, log = orc.reconstruct(cfg, sino, cfg)
    got, glog = orc.reconstruct_steps(cfg, sino, cfg)
    assert np.array_equal(got, want)
    assert np.array_equal(glog[:, 1], log[:, 1]) and np.allclose(glog, log, rtol=1e-12, atol=0)
