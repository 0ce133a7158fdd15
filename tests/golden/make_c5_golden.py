#!/usr/bin/env python
"""Writes tests/golden/c5_full_oracle.npz: the ORACLE's reconstruction of BASELINE.json configs[4]
(3D cone beam 512x512x128, 60 views x 384x512, 10 CGLS + 5 GD per outer iteration) at FULL size,
sampled, after every outer iteration reached. Calls only oracle/ and the seeded input generator
(ctr_inputs); nothing from the CUDA path. tests/test_gpu_cone.py compares ctr_reconstruct against it.

The full volume is 268 MB in fp64, so what is stored per checkpoint (outer iteration n) is
  samples[n]  the oracle image at N_SAMPLES seeded voxel positions (fp64),
  planes[n]   the L2 norm of every z-plane (128 values) and `norm[n]` of the whole volume,
  log         per sweep (sigma, Armijo k, E0, |g|^2) - what steers the iteration.
The outer loop is composed here from the oracle's own steps (orc.cgls, orc.update_weights,
orc.eptv_step, clamp) exactly as orc_reconstruct (O10) composes them, so that a
checkpoint can be written after every outer iteration of one long run;
tests/test_oracle_pins.py::test_composed_outer_loop_is_orc_reconstruct checks that this composition
gives orc_reconstruct's result bit for bit.

    python tests/golden/make_c5_golden.py [--n-outer 20] [--threads 6]

About 20 minutes per outer iteration on 8 cores. The file is rewritten (atomically) after every outer
iteration (checkpoints KEEP and the last one reached stay in it); a rerun continues from nothing (the oracle
has no warm start), so let it finish.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
ROOT = HERE.parent.parent
sys.path.insert(0, str(ROOT))

N_SAMPLES = 131072
SAMPLE_SEED = 10092288 + 5000 + 77
KEEP = (1, 2, 3, 5, 10, 15, 20)  # checkpoints kept in the file besides the last one reached (1 MB each)


def oracle_fingerprint() -> str:
    """sha256 of oracle/ctr_oracle.c with comments and white space removed: changes when its code does."""
    import re
    src = (ROOT / "oracle" / "ctr_oracle.c").read_text()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return hashlib.sha256("".join(src.split()).encode()).hexdigest()[:16]


def sample_positions(nvox: int) -> np.ndarray:
    return np.sort(np.random.Generator(np.random.PCG64(SAMPLE_SEED)).choice(nvox, N_SAMPLES, replace=False))


def composed_reconstruct(orc, cfg, sino, n_outer, on_outer=None):
    """O10 composed from the oracle's steps; on_outer(n, f, log) is called after outer iteration n."""
    f = np.zeros(cfg.img_shape if cfg.ndim == 3 else (1, cfg.ny, cfg.nx))
    log = []
    for it in range(n_outer):
        f = orc.cgls(cfg, sino, f, cfg.n_cgls).reshape(f.shape)           # Step 1 (:171)
        v = f.copy()
        for _ in range(cfg.n_gd):                                          # Step 2 (:172)
            w, sig = orc.update_weights(f, cfg.sigma_quantile, cfg.eps, cfg.weights_mode, ndim=cfg.ndim)
            f, k, e0, g2, _t = orc.eptv_step(f, v, w, cfg.lam, cfg, ndim=cfg.ndim)
            log.append((sig, k, e0, g2))
        if cfg.positivity:                                                 # Step 3 (:173)
            f = np.maximum(f, 0.0)
        if on_outer:
            on_outer(it + 1, f, np.array(log))
    return f, np.array(log)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n-outer", type=int, default=20)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--out", default=str(HERE / "c5_full_oracle.npz"))
    args = ap.parse_args()
    if args.threads:
        os.environ["OMP_NUM_THREADS"] = str(args.threads)
    from ctr_inputs import get_config, make_case
    from oracle import ctr_oracle as orc

    orc.build()
    cfg = get_config("c5")
    sino = make_case(cfg, raster=False)["sino"].astype(np.float64)
    pos = sample_positions(cfg.nx * cfg.ny * cfg.nz)
    store = {"positions": pos, "oracle_sha": np.array(oracle_fingerprint()), "n_cgls": cfg.n_cgls, "n_gd": cfg.n_gd}
    t0 = time.time()

    def on_outer(n, f, log):
        store[f"samples_{n}"] = f.ravel()[pos].copy()
        store[f"planes_{n}"] = np.sqrt((f.reshape(cfg.nz, -1) ** 2).sum(axis=1))
        store[f"norm_{n}"] = np.linalg.norm(f)
        store["log"] = log
        store["n_done"] = n
        if n - 1 not in KEEP:
            for key in ("samples", "planes", "norm"):
                store.pop(f"{key}_{n - 1}", None)
        tmp = args.out + f".tmp{os.getpid()}.npz"
        np.savez_compressed(tmp, **store)
        os.replace(tmp, args.out)
        print(f"outer {n}: {time.time() - t0:.0f} s, |f| = {store[f'norm_{n}']:.6e}, ks = {log[-cfg.n_gd:, 1].astype(int)}",
              flush=True)

    composed_reconstruct(orc, cfg, sino, args.n_outer, on_outer)


if __name__ == "__main__":
    main()
