"""GPU parity of the projector pair through the C ABI (ctr_forward / ctr_back) against the fp64
oracle, element by element on the same seeded inputs. Tolerance (north_star): relative L2 <= 1e-5
for one P or P^T application; adjoint identity <= 1e-5; the two kernels' matrices bit-identical."""
import math

import numpy as np
import pytest

from ctr_inputs import get_config, make_case, scaled_config
from ctr_inputs.configs import Config

pytestmark = pytest.mark.gpu

TOL_OP = 1e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def ctr():
    import paper_1009_2288_b200 as m
    m.load_library()
    return m


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b))


def assert_close(a, b, tol):
    """relative L2 error <= tol (north_star's norm) AND no single element further off than 10 tol of the largest
    reference value (30 tol for one operator application): a handful of wrong border pixels or one wrong view would
    hide under the L2 norm alone. Why 30: a ray almost parallel to a grid axis (slope m -> 0) splits its length in a
    slab between two neighbouring cells at a crossing whose position is known to ~1e-5 pixel in fp32, i.e. the split
    moves by ~1e-5 / |m| of the slab length; the SUM over the two cells is exact, single elements of P^T y differ by up
    to ~2e-4 of the largest value at 512^2 (measured)."""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    err_l2 = float(np.linalg.norm(a - b) / np.linalg.norm(b))
    err_max = float(np.max(np.abs(a - b)) / np.max(np.abs(b)))
    assert err_l2 <= tol, (err_l2, tol)
    elem = (30 if tol <= 2e-5 else 10) * tol
    assert err_max <= elem, (err_max, elem)


def gpu_forward(ctr, torch, cfg, img, flags=0):
    h = ctr.ctr_create(cfg, flags=flags)
    x = torch.from_numpy(np.ascontiguousarray(img, dtype=np.float32)).cuda()
    y = torch.full(h.sino_shape, float("nan"), dtype=torch.float32, device="cuda")
    h.ctr_forward(x, y)
    torch.cuda.synchronize()
    h.close()
    return y.cpu().numpy()


def gpu_back(ctr, torch, cfg, sino, flags=0):
    h = ctr.ctr_create(cfg, flags=flags)
    y = torch.from_numpy(np.ascontiguousarray(sino, dtype=np.float32)).cuda()
    x = torch.full(h.img_shape, float("nan"), dtype=torch.float32, device="cuda")
    h.ctr_back(y, x)
    torch.cuda.synchronize()
    h.close()
    return x.cpu().numpy()


def odd2d(**kw):
    base = dict(name="odd", index=92, ndim=2, nx=37, ny=29, nz=1, dx=1.3, dy=0.9, dz=1.0, nviews=17, nu=53,
                nv=1, du=1.7, dv=1.0, dso=300.0, dsd=520.0, cx=1.1, cy=-2.3, u_off=0.4, theta0=0.1)
    base.update(kw)
    return Config(**base)


@pytest.mark.parametrize("name", ["c1", "c2", "c3"])
def test_forward_and_back_match_oracle(ctr, torch_cuda, orc, name):
    cfg = get_config(name)
    case = make_case(cfg)
    truth, sino = case["truth"][0], case["sino"][0]
    got = gpu_forward(ctr, torch_cuda, cfg, truth[None])[0]
    want = orc.forward(cfg, truth.astype(np.float64))
    assert_close(got, want, TOL_OP)
    got = gpu_back(ctr, torch_cuda, cfg, sino[None])[0]
    want = orc.back(cfg, sino.astype(np.float64))
    assert_close(got, want, TOL_OP)


@pytest.mark.parametrize("cfg", [odd2d(), odd2d(det_type=1, du=1.0), odd2d(nx=1, ny=1, dx=5.0, dy=5.0),
                                 odd2d(nviews=8, nu=11, theta0=0.0, cx=0.0, cy=0.0, u_off=0.0)],
                         ids=["ragged", "arc", "single-pixel", "axis-parallel"])
def test_odd_geometries_random_inputs(ctr, torch_cuda, orc, cfg):
    """Ragged sizes (not multiples of any tile), off-centre grid, detector shift, arc detector,
    rays exactly parallel to an axis (odd nu, theta = 0/90/...). Random (rough) inputs."""
    rng = np.random.default_rng(21)
    x = rng.random((1, cfg.ny, cfg.nx)).astype(np.float32)
    y = rng.random((1, cfg.nviews, cfg.nu)).astype(np.float32)
    assert_close(gpu_forward(ctr, torch_cuda, cfg, x)[0], orc.forward(cfg, x[0].astype(np.float64)), 2e-5)
    assert_close(gpu_back(ctr, torch_cuda, cfg, y)[0], orc.back(cfg, y[0].astype(np.float64)), 2e-5)


def test_batched_slices_match_oracle_per_slice(ctr, torch_cuda, orc):
    """V = 4 internal layout with a ragged batch (6 = 4 + 2) on the c2 geometry."""
    cfg = scaled_config("c2", batch=6)
    case = make_case(cfg)
    got_s = gpu_forward(ctr, torch_cuda, cfg, case["truth"])
    got_i = gpu_back(ctr, torch_cuda, cfg, case["sino"])
    assert got_s.shape == (6, cfg.nviews, cfg.nu) and got_i.shape == (6, cfg.ny, cfg.nx)
    for sl in (0, 3, 5):
        assert_close(got_s[sl], orc.forward(cfg, case["truth"][sl].astype(np.float64)), TOL_OP)
        assert_close(got_i[sl], orc.back(cfg, case["sino"][sl].astype(np.float64)), TOL_OP)
    # batched vs single-slice operators: same p_ij bit for bit, added in different fixed orders (ctr_si.cu,
    # ctr_ell.cuh), so they agree to fp32 rounding
    one = scaled_config("c2", batch=1)
    assert_close(gpu_forward(ctr, torch_cuda, one, case["truth"][4:5])[0], got_s[4].astype(np.float64), 1e-6)
    assert_close(gpu_back(ctr, torch_cuda, one, case["sino"][4:5])[0], got_i[4].astype(np.float64), 1e-6)


@pytest.mark.parametrize("name,batch", [("c1", 1), ("c3", 1), ("c2", 5)])
def test_adjoint_identity_on_gpu(ctr, torch_cuda, name, batch):
    """PAPER.md:471 (A3'): <Px,y> = <x,P^T y> to fp32 rounding (dots accumulated in fp64)."""
    cfg = scaled_config(name, batch=batch)
    rng = np.random.default_rng(22)
    x = rng.random((batch, cfg.ny, cfg.nx)).astype(np.float32)
    y = rng.random((batch, cfg.nviews, cfg.nu)).astype(np.float32)
    px = gpu_forward(ctr, torch_cuda, cfg, x).astype(np.float64)
    pty = gpu_back(ctr, torch_cuda, cfg, y).astype(np.float64)
    for sl in range(batch):
        lhs, rhs = (px[sl] * y[sl]).sum(), (x[sl] * pty[sl]).sum()
        assert abs(lhs - rhs) <= TOL_OP * np.linalg.norm(px[sl]) * np.linalg.norm(y[sl])
        assert abs(lhs - rhs) <= 2e-6 * abs(lhs)


def test_forward_and_back_use_bit_identical_matrices(ctr, torch_cuda, orc):
    """Exact transpose: probing P with unit images and P^T with unit sinograms gives the same
    matrix bit for bit, and it equals the oracle's dense matrix to fp32 accuracy."""
    cfg = odd2d(nx=9, ny=7, nviews=6, nu=14, dx=2.0, dy=1.5)
    npix, nray = cfg.nx * cfg.ny, cfg.nviews * cfg.nu
    torch = torch_cuda
    h = ctr.ctr_create(cfg)
    A_f = np.zeros((nray, npix), np.float32)
    A_b = np.zeros((nray, npix), np.float32)
    x = torch.zeros(h.img_shape, device="cuda")
    y = torch.zeros(h.sino_shape, device="cuda")
    for j in range(npix):
        x.zero_()
        x.view(-1)[j] = 1.0
        h.ctr_forward(x, y)
        A_f[:, j] = y.view(-1).cpu().numpy()
    for r in range(nray):
        y.zero_()
        y.view(-1)[r] = 1.0
        h.ctr_back(y, x)
        A_b[r, :] = x.view(-1).cpu().numpy()
    h.close()
    assert np.array_equal(A_f, A_b)
    A = orc.matrix(cfg)
    assert np.max(np.abs(A_f - A)) <= 2e-5 * A.max()
    assert ((A_f > 0) == (A > 1e-4)).mean() > 0.98


def test_zero_and_linearity(ctr, torch_cuda):
    cfg = get_config("c1")
    z = gpu_forward(ctr, torch_cuda, cfg, np.zeros((1, cfg.ny, cfg.nx), np.float32))
    assert np.all(z == 0)
    zb = gpu_back(ctr, torch_cuda, cfg, np.zeros((1, cfg.nviews, cfg.nu), np.float32))
    assert np.all(zb == 0)


def test_invalid_arguments(ctr, torch_cuda):
    torch = torch_cuda
    with pytest.raises(ctr.CtrError) as e:
        ctr.ctr_create(scaled_config("c1", dsd=100.0))      # dsd <= dso
    assert e.value.status == -1
    with pytest.raises(ctr.CtrError) as e:
        ctr.ctr_create(scaled_config("c1", dso=40.0, dsd=949.0))  # source inside the image circle
    assert e.value.status == -2
    h = ctr.ctr_create(get_config("c1"))
    x = torch.zeros(h.img_shape, device="cuda")
    b = torch.zeros(h.sino_shape, device="cuda")
    with pytest.raises(ctr.CtrError):
        h.ctr_cgls(b, x, -1)
    with pytest.raises(ctr.CtrError):
        h.ctr_update_weights(x, torch.zeros(h.w_shape, device="cuda"), quantile=0.0)
    with pytest.raises(ValueError):
        h.ctr_forward(x, torch.zeros(3, device="cuda"))
    mis = torch.zeros(h.n_img + 1, device="cuda")[1:]        # 4-byte aligned only
    rc = h._L.ctr_forward(h._h, mis.data_ptr(), b.data_ptr(), None)
    assert rc == -1
    x0 = x.clone()
    h.ctr_cgls(b, x, 0)                                      # n_iter = 0: no-op
    torch.cuda.synchronize()
    assert torch.equal(x, x0)
    h.close()


# ------------------------------------------------------------------ the bench configuration itself
def test_c4_full_batch_operators_and_cgls(ctr, torch_cuda, orc):
    """configs[3] as bench.py launches it: 64 slices (LQ = 16, hit-table gather). P, P^T and three CGLS
    iterations on all 64 slices in one call; slices 0, 21 and 63 are compared with the oracle one by one,
    the adjoint identity is checked on every slice."""
    torch = torch_cuda
    cfg = get_config("c4")
    assert cfg.batch == 64
    rng = np.random.default_rng(404)
    x = rng.random((64, cfg.ny, cfg.nx), dtype=np.float32)
    y = rng.random((64, cfg.nviews, cfg.nu), dtype=np.float32)
    # slice 21: a structured image (disc + ramp) rather than noise
    jj, ii = np.mgrid[0:cfg.ny, 0:cfg.nx]
    x[21] = (0.019 * (((ii - 260) ** 2 + (jj - 240) ** 2) < 200 ** 2) + 1e-5 * ii).astype(np.float32)
    h = ctr.ctr_create(cfg)
    xg, yg = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    Px = torch.full(h.sino_shape, float("nan"), device="cuda")
    Pty = torch.full(h.img_shape, float("nan"), device="cuda")
    h.ctr_forward(xg, Px)
    h.ctr_back(yg, Pty)
    u = torch.zeros(h.img_shape, device="cuda")
    u[21] = 0.01
    h.ctr_cgls(Px, u, 3)                      # consistent data: b = P x
    torch.cuda.synchronize()
    lhs = (Px.double() * yg.double()).sum(dim=(1, 2))
    rhs = (xg.double() * Pty.double()).sum(dim=(1, 2))
    nrm = Px.double().flatten(1).norm(dim=1) * yg.double().flatten(1).norm(dim=1)
    assert float(((lhs - rhs).abs() / nrm).max()) <= 1e-5
    Px, Pty, u = Px.cpu().numpy(), Pty.cpu().numpy(), u.cpu().numpy()
    h.close()
    for sl in (0, 21, 63):
        want_s = orc.forward(cfg, x[sl].astype(np.float64))
        assert_close(Px[sl], want_s, TOL_OP)
        assert_close(Pty[sl], orc.back(cfg, y[sl].astype(np.float64)), TOL_OP)
        x0 = np.full((cfg.ny, cfg.nx), 0.01 if sl == 21 else 0.0)
        assert_close(u[sl], orc.cgls(cfg, Px[sl].astype(np.float64), x0, 3), 1e-4)


@pytest.mark.parametrize("batch", [2, 20, 70])
def test_sub_warp_widths(ctr, torch_cuda, orc, batch):
    """batch 2 -> LQ = 1 (32 rays per warp); 20 -> LQ = 8; 70 -> 18 quads -> LQ = 16, two super-groups, the
    second mostly padding."""
    cfg = scaled_config("c1", batch=batch)
    rng = np.random.default_rng(405)
    x = rng.random((batch, cfg.ny, cfg.nx), dtype=np.float32)
    y = rng.random((batch, cfg.nviews, cfg.nu), dtype=np.float32)
    got_s = gpu_forward(ctr, torch_cuda, cfg, x)
    got_i = gpu_back(ctr, torch_cuda, cfg, y)
    for sl in sorted({0, min(63, batch - 1), min(64, batch - 1), batch - 1}):
        assert_close(got_s[sl], orc.forward(cfg, x[sl].astype(np.float64)), TOL_OP)
        assert_close(got_i[sl], orc.back(cfg, y[sl].astype(np.float64)), TOL_OP)


# ------------------------------------------------------------------ stored matrices (single slice)
def _both_ways(ctr, torch, cfg, x, y):
    """(P x, P^T y) with the stored sliced-ELL matrices and with the on-the-fly kernels."""
    out = []
    for flags in (0, ctr.CTR_GEOM_NO_TABLES):
        out.append((gpu_forward(ctr, torch, cfg, x, flags), gpu_back(ctr, torch, cfg, y, flags)))
    return out


@pytest.mark.parametrize("cfg", [get_config("c2"), odd2d(), odd2d(det_type=1, du=1.0)], ids=["c2", "odd", "arc"])
def test_stored_matrices_equal_on_the_fly_kernels(ctr, torch_cuda, cfg):
    """The lookup-table operators hold the very values the on-the-fly kernels compute. P^T adds
    them in the same order (identical bits); the stored P of a 2D slice splits every ray over 16 threads, so its
    sums agree with the on-the-fly kernel to fp32 rounding."""
    rng = np.random.default_rng(406)
    x = rng.random((1, cfg.ny, cfg.nx), dtype=np.float32)
    y = rng.random((1, cfg.nviews, cfg.nu), dtype=np.float32)
    (s_tab, i_tab), (s_fly, i_fly) = _both_ways(ctr, torch_cuda, cfg, x, y)
    assert_close(s_tab, s_fly.astype(np.float64), 1e-6)
    assert np.array_equal(i_tab, i_fly)


def test_batched_gather_fallback_matches_quad_table(ctr, torch_cuda):
    """batch > 1: the on-the-fly gather k_si_back (used when the quad hit table cannot be allocated) against
    the table-driven k_si_back_quad: same p_ij, different fixed summation orders."""
    cfg = scaled_config("c2", batch=9)
    y = np.random.default_rng(407).random((9, cfg.nviews, cfg.nu), dtype=np.float32)
    (_, i_tab), (_, i_fly) = _both_ways(ctr, torch_cuda, cfg, np.zeros((9, cfg.ny, cfg.nx), np.float32), y)
    assert_close(i_tab, i_fly.astype(np.float64), 1e-6)


@pytest.mark.parametrize("batch", [5, 64, 70])
def test_batched_stored_P_equals_on_the_fly_P(ctr, torch_cuda, batch):
    """NEXT-2 for batches ("save the projection matrix ... as a lookup table"): the stored P shared by
    all slices (k_si_forward_tab, a sparse-matrix x dense-matrix product over the slices) holds the entries the
    on-the-fly kernel k_si_forward computes and adds them in the same order: identical bits."""
    cfg = scaled_config("c2", batch=batch)
    x = np.random.default_rng(408).random((batch, cfg.ny, cfg.nx), dtype=np.float32)
    h = ctr.ctr_create(cfg)
    assert h.ctr_path_info()["forward"] == "k_si_forward_tab"
    h.close()
    s_tab = gpu_forward(ctr, torch_cuda, cfg, x)
    s_fly = gpu_forward(ctr, torch_cuda, cfg, x, ctr.CTR_GEOM_NO_STORED_P)
    assert np.array_equal(s_tab, s_fly)


# ------------------------------------------------------------------ NEXT-1: the paper's backprojector Eq. (11)
def gpu_back_pixel(ctr, torch, cfg, sino):
    h = ctr.ctr_create(cfg)
    y = torch.from_numpy(np.ascontiguousarray(sino, dtype=np.float32)).cuda()
    x = torch.full(h.img_shape, float("nan"), dtype=torch.float32, device="cuda")
    h.ctr_back_pixel(y, x)
    torch.cuda.synchronize()
    h.close()
    return x.cpu().numpy()


@pytest.mark.parametrize("cfg,batch", [(get_config("c2"), 1), (odd2d(), 1), (odd2d(det_type=1, du=1.0), 3),
                                       (scaled_config("c1", batch=11), 11)], ids=["c2", "odd", "arc3", "c1x11"])
def test_back_pixel_eq11_matches_oracle(ctr, torch_cuda, orc, cfg, batch):
    """ctr_back_pixel (Eq. 11) against orc.back_eq11 on random sinograms (the hardest input
    for an interpolating operator), relative L2 <= 1e-5 as for the other operators."""
    if cfg.batch != batch:
        cfg = Config(**{**cfg.__dict__, "batch": batch})
    y = np.random.default_rng(408).random((batch, cfg.nviews, cfg.nu), dtype=np.float32)
    got = gpu_back_pixel(ctr, torch_cuda, cfg, y)
    for sl in sorted({0, batch // 2, batch - 1}):
        assert_close(got[sl], orc.back_eq11(cfg, y[sl].astype(np.float64)), TOL_OP)


def test_back_pixel_adjoint_mismatch_below_one_percent_on_gpu(ctr, torch_cuda):
    """The paper's printed number on the CUDA path: <f, Eq11(y)> vs <ctr_forward(f), y> on the
    paper's scanner geometry (arc detector, :217) with smooth f and y."""
    cfg = Config(name="paper", index=91, ndim=2, nx=512, ny=512, nz=1, dx=500.0 / 512, dy=500.0 / 512, dz=1.0,
                 nviews=40, nu=888, nv=1, du=1.0239, dv=1.0, dso=541.0, dsd=949.075, det_type=1)
    jj, ii = np.mgrid[0:512, 0:512]
    f = np.exp(-(((ii - 300) * 0.9766) ** 2 + ((jj - 230) * 0.9766) ** 2) / (2 * 40.0 ** 2)).astype(np.float32)[None]
    kk, bb = np.mgrid[0:cfg.nviews, 0:cfg.nu]
    y = (1.0 + 0.5 * np.cos(2 * np.pi * kk / cfg.nviews) * np.cos(3.0 * (bb / cfg.nu - 0.5))).astype(np.float32)[None]
    Pf = gpu_forward(ctr, torch_cuda, cfg, f).astype(np.float64)
    Bty = gpu_back_pixel(ctr, torch_cuda, cfg, y).astype(np.float64)
    lhs, rhs = float((f * Bty).sum()), float((Pf * y).sum())
    assert 1e-9 * abs(rhs) < abs(lhs - rhs) <= 0.01 * abs(rhs)


@pytest.mark.parametrize("batch", [1, 5])
def test_arc_detector_and_explicit_angles(ctr, torch_cuda, orc, batch):
    """The paper's detector type (ARC) with an explicit, non-uniform angle list (ctr_geometry.angles)
    and an off-centre grid: single slice (stored matrices) and batched (slice-interleaved) operators."""
    ang = [0.05, 0.9, 1.7, 2.2, 3.3, 4.1, 4.15, 5.9]
    base = odd2d(det_type=1, du=1.0, nviews=len(ang), batch=batch)
    geo = dict(base.geometry_dict(), angles=ang)
    rng = np.random.default_rng(409)
    x = rng.random((batch, base.ny, base.nx), dtype=np.float32)
    y = rng.random((batch, base.nviews, base.nu), dtype=np.float32)
    got_s = gpu_forward(ctr, torch_cuda, geo, x)
    got_i = gpu_back(ctr, torch_cuda, geo, y)
    one = dict(geo, batch=1)
    for sl in {0, batch - 1}:
        assert_close(got_s[sl], orc.forward(one, x[sl].astype(np.float64)), TOL_OP)
        assert_close(got_i[sl], orc.back(one, y[sl].astype(np.float64)), TOL_OP)
    # and the angles really were used: a uniform scan gives a different sinogram
    assert rel(gpu_forward(ctr, torch_cuda, base, x)[0], got_s[0].astype(np.float64)) > 1e-2


def _random_geometry(rng, batch):
    """A seeded random scanner: ragged sizes, anisotropic pixels, off-centre grid, shifted detector, either detector type,
    source and detector outside the grid's circumscribed circle."""
    nx, ny = int(rng.integers(1, 70)), int(rng.integers(1, 70))
    dx, dy = float(rng.uniform(0.6, 2.0)), float(rng.uniform(0.6, 2.0))
    cx, cy = float(rng.uniform(-3, 3)), float(rng.uniform(-3, 3))
    rad = math.hypot(abs(cx) + 0.5 * nx * dx + dx, abs(cy) + 0.5 * ny * dy + dy)
    dso = rad * float(rng.uniform(1.3, 6.0))
    dsd = dso + rad * float(rng.uniform(1.3, 4.0))
    return Config(name="fuzz", index=94, ndim=2, nx=nx, ny=ny, nz=1, dx=dx, dy=dy, dz=1.0,
                  nviews=int(rng.integers(1, 40)), nu=int(rng.integers(1, 120)), nv=1,
                  du=float(rng.uniform(0.5, 3.0)) * dsd / dso, dv=1.0, dso=dso, dsd=dsd, cx=cx, cy=cy,
                  u_off=float(rng.uniform(-2, 2)), theta0=float(rng.uniform(0, 6.28)),
                  det_type=int(rng.integers(0, 2)), batch=batch)


@pytest.mark.parametrize("seed", range(12))
def test_random_geometries_against_oracle(ctr, torch_cuda, orc, seed):
    """Seeded random geometries and batch sizes (compute-sanitizer is closed on this pool: ragged sizes against the
    oracle are the memory-safety net): P and P^T within 2e-5 of the oracle on rough random inputs (first and last slice),
    tables against on-the-fly kernels, and the adjoint identity on the device."""
    rng = np.random.default_rng(1000 + seed)
    batch = int(rng.choice([1, 1, 2, 3, 5, 9, 17, 33]))
    cfg = _random_geometry(rng, batch)
    one = Config(**{**cfg.__dict__, "batch": 1})
    x = rng.random((batch, cfg.ny, cfg.nx)).astype(np.float32)
    y = rng.random((batch, cfg.nviews, cfg.nu)).astype(np.float32)
    (s_tab, i_tab), (s_fly, i_fly) = _both_ways(ctr, torch_cuda, cfg, x, y)
    for sl in sorted({0, batch - 1}):
        want_s, want_i = orc.forward(one, x[sl].astype(np.float64)), orc.back(one, y[sl].astype(np.float64))
        if np.linalg.norm(want_s) > 0:
            assert_close(s_tab[sl], want_s, 2e-5)
            assert_close(s_fly[sl], want_s, 2e-5)
        else:
            assert not s_tab[sl].any() and not s_fly[sl].any()
        if np.linalg.norm(want_i) > 0:
            assert_close(i_tab[sl], want_i, 2e-5)
            assert_close(i_fly[sl], want_i, 2e-5)
        else:
            assert not i_tab[sl].any() and not i_fly[sl].any()
    lhs = float((s_tab.astype(np.float64) * y).sum())
    rhs = float((x.astype(np.float64) * i_tab).sum())
    assert abs(lhs - rhs) <= 1e-5 * (np.linalg.norm(s_tab.astype(np.float64)) * np.linalg.norm(y.astype(np.float64)) + 1e-30)
