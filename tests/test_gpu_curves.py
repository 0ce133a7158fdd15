"""NEXT-3: convergence curves of EP-TV against plain TV and against restarted CGLS alone on the
synthetic c2 workload, like the paper's Fig. 4, with the paper's metrics Eq. 12-14
(ctr_inputs/metrics.py). The CUDA path is run one outer iteration at a time (warm_start, which continues the iteration
bit for bit: tests/test_gpu_solvers.py); the end points are compared with the oracle's full runs.

No quality claim is tested: the paper tuned lambda and the sigma percentage by hand per data set (:110, :175). What is
asserted is what must hold for any setting: every curve starts at the first CGLS result, all errors stay finite and
below the zero image's, plain TV with the same lambda smooths more (lower TV energy of the result), and the curves'
end points are the oracle's. The table the run prints is kept in profiles/r2_convergence_c2.md."""
import numpy as np
import pytest

from ctr_inputs import get_config, make_case, scaled_config
from ctr_inputs.metrics import edge_cross_correlation, relative_error, snr_db

pytestmark = pytest.mark.gpu


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


def _curve(ctr, torch, cfg, sino, truth, **over):
    h = ctr.ctr_create(cfg)
    img = torch.zeros(h.img_shape, device="cuda")
    y = torch.from_numpy(sino).cuda()
    rows = []
    roi = (slice(cfg.ny // 2 - 8, cfg.ny // 2 + 8), slice(cfg.nx // 2 - 8, cfg.nx // 2 + 8))  # inside the body ellipse
    for it in range(cfg.n_outer):
        h.ctr_reconstruct(y, img, ctr.make_params(cfg, n_outer=1, warm_start=int(it > 0), **over))
        torch.cuda.synchronize()
        f = img.cpu().numpy()[0].astype(np.float64)
        rows.append((relative_error(f, truth), edge_cross_correlation(f, truth), snr_db(f, roi)))
    h.close()
    return np.array(rows), f


def test_convergence_curves_eptv_tv_cgls_on_c2(ctr, torch_cuda, orc):
    torch = torch_cuda
    cfg = get_config("c2")
    case = make_case(cfg)
    sino, truth = case["sino"], case["truth"][0].astype(np.float64)
    runs = {"EP-TV": dict(weights_mode=0), "TV": dict(weights_mode=1), "CGLS only": dict(n_gd=0)}
    curves, finals = {}, {}
    for name, over in runs.items():
        c = scaled_config("c2", **over) if "n_gd" in over else cfg
        curves[name], finals[name] = _curve(ctr, torch, c, sino, truth, **over)
    print("\n[curves] c2 (256^2, 40 views, I0 = 5e3, lambda = 0.02, q = 0.90), Eq. 12 relative error / Eq. 13 edge "
          "cross-correlation / Eq. 14 SNR (dB, 16x16 ROI at the centre) after outer iteration n")
    print("  n   " + "".join(f"{k:>32s}" for k in runs))
    for it in range(cfg.n_outer):
        print(f"  {it + 1:2d}  " + "".join(f"   {curves[k][it, 0]:8.5f} / {curves[k][it, 1]:5.3f} / {curves[k][it, 2]:6.2f}" for k in runs))
    zero_err = relative_error(np.zeros_like(truth), truth)
    for k, c in curves.items():
        assert np.isfinite(c).all() and (c[:, 0] < zero_err).all(), k
    # plain TV (w = 1 >= the EP-TV weights) regularises more: its result has the smaller total variation
    tv_of = lambda f: np.abs(np.diff(f, axis=0)).sum() + np.abs(np.diff(f, axis=1)).sum()
    assert tv_of(finals["TV"]) < tv_of(finals["EP-TV"]) < tv_of(finals["CGLS only"])
    # end points against the oracle's full schedules
    for name, over in (("EP-TV", {}), ("TV", dict(weights_mode=1))):
        c = scaled_config("c2", **over)
        want, _, _ = orc.reconstruct(c, sino[0].astype(np.float64), c)
        err = np.linalg.norm(finals[name] - want) / np.linalg.norm(want)
        assert err <= 1e-3, (name, err)
