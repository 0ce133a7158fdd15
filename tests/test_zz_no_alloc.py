"""ctr_forward_noalloc (include/ctr.h): the forward projector for callers that cannot allocate - no handle, no
cudaMalloc, its scratch (ray table + transposed image copy) in one file-scope device array of fixed size - against the
existing path ctr_forward, on calls in a row that share that array. Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from ctr_inputs import get_config, scaled_config
from ctr_inputs.configs import Config

pytestmark = pytest.mark.gpu

TOL_OP = 1e-5   # north_star: one P application, relative L2 (tests/test_gpu_operators.py)


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


def assert_close(a, b, tol):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    assert float(np.linalg.norm(a - b) / np.linalg.norm(b)) <= tol
    assert float(np.max(np.abs(a - b)) / np.max(np.abs(b))) <= 30 * tol


def handle_forward(ctr, torch, cfg, x, flags=0):
    h = ctr.ctr_create(cfg, flags=flags)
    sino = torch.full(h.sino_shape, float("nan"), device="cuda")
    h.ctr_forward(x, sino)
    torch.cuda.synchronize()
    h.close()
    return sino.cpu().numpy()[0]


def test_forward_noalloc_matches_ctr_forward_on_calls_in_a_row(ctr, torch_cuda, orc):
    torch = torch_cuda
    rng = np.random.default_rng(77)
    ragged = Config(name="odd", index=96, ndim=2, nx=37, ny=29, nz=1, dx=1.3, dy=0.9, dz=1.0, nviews=17, nu=53, nv=1,
                    du=1.0, dv=1.0, dso=300.0, dsd=520.0, cx=1.1, cy=-2.3, u_off=0.4, theta0=0.1, det_type=1)
    cfgs = [scaled_config("c2", batch=1), ragged, scaled_config("c3", batch=1), scaled_config("c2", batch=1)]
    xs = [torch.from_numpy(rng.random((1, c.ny, c.nx), dtype=np.float32)).cuda() for c in cfgs]
    xs[3] = xs[0]                                               # the fourth call repeats the first
    outs = [torch.full((1, c.nviews, c.nu), float("nan"), device="cuda") for c in cfgs]
    ctr.ctr_forward_noalloc(cfgs[1], xs[1], outs[1])            # warm-up: kernels loaded, the array's address looked up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for c, x, o in zip(cfgs, xs, outs):                         # four calls in a row on one stream, no sync in between:
        ctr.ctr_forward_noalloc(c, x, o)                        # each finds the scratch as the previous call left it
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                # nothing was allocated on the device
    got = [o.cpu().numpy()[0] for o in outs]
    for c, x, g in zip(cfgs[:3], xs[:3], got[:3]):
        assert np.isfinite(g).all()
        # the existing path: on the fly (same kernels: identical bits) and with its lookup tables (fp32 rounding)
        assert np.array_equal(g, handle_forward(ctr, torch, c, x, ctr.CTR_GEOM_NO_TABLES))
        assert_close(g, handle_forward(ctr, torch, c, x), TOL_OP)
    assert np.array_equal(got[3], got[0])                       # nothing of the calls in between leaked into the result
    assert_close(got[0], orc.forward(cfgs[0], xs[0].cpu().numpy()[0].astype(np.float64)), TOL_OP)


def test_forward_noalloc_rejects_what_does_not_fit(ctr, torch_cuda):
    torch = torch_cuda
    big = scaled_config("c3", batch=1, nx=1024, ny=512)          # 2 x the pixels the fixed scratch holds
    many = scaled_config("c3", batch=1, nu=1200)                 # 72 000 rays > 65 536
    x = torch.zeros((1, 512, 1024), device="cuda")
    y = torch.full((1, 60, 1200), 7.0, device="cuda")
    for cfg, xi, yi in ((big, x, y[:, :, :888].contiguous()), (many, x[:, :, :512].contiguous(), y)):
        with pytest.raises(ctr.CtrError) as e:
            ctr.ctr_forward_noalloc(cfg, xi, yi)
        assert e.value.status == ctr.binding.CTR_ETOOBIG and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert float(y.min()) == 7.0                                 # nothing was enqueued
    with pytest.raises(ctr.CtrError) as e:                       # batches and explicit angle lists need a handle
        ctr.ctr_forward_noalloc(scaled_config("c1", batch=2), torch.zeros((2, 64, 64), device="cuda")[:1].contiguous(),
                                torch.zeros((1, 30, 96), device="cuda"))
    assert e.value.status == ctr.binding.CTR_EINVAL
