"""Seeded ellipse / ellipsoid phantoms, their analytic sinograms, noise and rasters.

Stand-ins for the paper's NCAT / chest / Catphan data,
which are not available; the layouts are this repo's own.
Everything is numpy fp64 and deterministic given (config, slice):
    seed = 10092288 + 1000*config.index + slice          (numpy PCG64)

The sinogram is the ANALYTIC line integral of the ellipses along each source ->
detector-bin line (no pixel grid involved), so it also serves as an independent
check of the oracle's projector (tests/test_oracle_pins.py, pin (iii)).
Ray convention (App. III A6: ray direction (cos(beta+theta), sin(beta+theta))):
    source  S_k = -dso (cos th_k, sin th_k, 0)
    centre  C_k = (dsd-dso) (cos th_k, sin th_k, 0)
    e_u = (-sin th_k, cos th_k, 0),  e_v = (0,0,1)
    flat:   D = C_k + t_a e_u + v_b e_v,  t_a = (a-(nu-1)/2+u_off) du,  v_b = (b-(nv-1)/2+v_off) dv
    arc:    direction angle th_k + t_a/dsd, at distance dsd from the source.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

from .configs import Config

MU_WATER = 0.019  # mm^-1


@dataclass(frozen=True)
class Ellipse:
    """Additive ellipse (2D: c ignored) / ellipsoid rotated by phi about z."""
    x: float
    y: float
    z: float
    a: float
    b: float
    c: float
    phi: float
    dmu: float


def _seed(cfg: Config, slice_index: int) -> int:
    return 10092288 + 1000 * cfg.index + slice_index


def _rng(cfg: Config, slice_index: int, stream: int = 0) -> np.random.Generator:
    # stream 0: phantom shape, stream 1: noise (so noise does not depend on the shape draws)
    ss = np.random.SeedSequence([_seed(cfg, slice_index), stream])
    return np.random.Generator(np.random.PCG64(ss))


def _inside_ellipse(rng, a, b, frac):
    r = frac * math.sqrt(rng.uniform())
    t = rng.uniform(0.0, 2.0 * math.pi)
    return a * r * math.cos(t), b * r * math.sin(t)


def _chest2d(rng, scale: float):
    s = scale
    ell = [Ellipse(0, 0, 0, 110 * s, 75 * s, math.inf, 0.0, MU_WATER),
           Ellipse(45 * s, 0, 0, 32 * s, 50 * s, math.inf, 0.0, -0.015),
           Ellipse(-45 * s, 0, 0, 32 * s, 50 * s, math.inf, 0.0, -0.015)]
    for m in range(12):
        x, y = _inside_ellipse(rng, 110 * s, 75 * s, 0.8)
        a = rng.uniform(3, 12) * s
        b = rng.uniform(3, 12) * s
        phi = rng.uniform(0, math.pi)
        dmu = rng.uniform(0.010, 0.020) if m < 4 else rng.uniform(-0.002, 0.002)
        ell.append(Ellipse(x, y, 0, a, b, math.inf, phi, dmu))
    return ell


def make_phantom(cfg: Config, slice_index: int = 0) -> list[Ellipse]:
    rng = _rng(cfg, slice_index, 0)
    kind = cfg.phantom
    if kind == "c1":
        ell = []
        for _ in range(6):
            r = 20.0 * math.sqrt(rng.uniform())
            t = rng.uniform(0, 2 * math.pi)
            ell.append(Ellipse(r * math.cos(t), r * math.sin(t), 0, rng.uniform(5, 16),
                               rng.uniform(5, 16), math.inf, rng.uniform(0, math.pi),
                               rng.uniform(0.002, 0.0066)))
        ell.append(Ellipse(10, 0, 0, 4, 4, math.inf, 0, 0.01 * MU_WATER))
        ell.append(Ellipse(-10, 0, 0, 6, 6, math.inf, 0, 0.01 * MU_WATER))
        return ell
    if kind == "chest":
        return _chest2d(rng, 1.0)
    if kind == "chest1.6":
        return _chest2d(rng, 1.6)
    if kind == "catphan":
        ell = [Ellipse(0, 0, 0, 100, 100, math.inf, 0, MU_WATER)]
        diam = [2, 3, 4, 5, 6, 8, 10, 12, 15]
        contrast = [0.003, 0.005, 0.01]
        for m, d in enumerate(diam):
            t = math.radians(40.0 * m)
            ell.append(Ellipse(40 * math.cos(t), 40 * math.sin(t), 0, d / 2, d / 2, math.inf, 0,
                               contrast[m % 3] * MU_WATER))
        for m, dmu in enumerate([-0.019, 0.019, 0.006, -0.006]):
            t = math.radians(45.0 + 90.0 * m)
            ell.append(Ellipse(75 * math.cos(t), 75 * math.sin(t), 0, 6, 6, math.inf, 0, dmu))
        return ell
    if kind == "chest3d":
        ell = [Ellipse(0, 0, 0, 120, 85, 200, 0, MU_WATER),
               Ellipse(50, 0, 0, 35, 50, 45, 0, -0.015),
               Ellipse(-50, 0, 0, 35, 50, 45, 0, -0.015)]
        for m in range(10):
            x, y = _inside_ellipse(rng, 120, 85, 0.75)
            z = rng.uniform(-35, 35)
            r = rng.uniform(5, 10)
            ell.append(Ellipse(x, y, z, r, r, r, 0, (0.01 if m % 2 == 0 else -0.01) * MU_WATER))
        for m in range(6):
            x, y = _inside_ellipse(rng, 120, 85, 0.8)
            z = rng.uniform(-40, 40)
            ell.append(Ellipse(x, y, z, rng.uniform(4, 12), rng.uniform(4, 12), rng.uniform(8, 30),
                               rng.uniform(0, math.pi), rng.uniform(0.010, 0.020)))
        return ell
    raise ValueError(f"unknown phantom recipe {kind!r}")


def view_angles(cfg: Config) -> np.ndarray:
    return cfg.theta0 + cfg.dtheta * np.arange(cfg.nviews, dtype=np.float64)


def ray_endpoints(cfg: Config, view: int):
    """Source S (3,) and detector points D (nv, nu, 3) of one view, fp64, mm."""
    th = cfg.theta0 + cfg.dtheta * view
    c, s = math.cos(th), math.sin(th)
    S = np.array([-cfg.dso * c, -cfg.dso * s, 0.0])
    t = (np.arange(cfg.nu) - (cfg.nu - 1) / 2.0 + cfg.u_off) * cfg.du
    v = (np.arange(cfg.nv) - (cfg.nv - 1) / 2.0 + cfg.v_off) * cfg.dv
    D = np.empty((cfg.nv, cfg.nu, 3))
    if cfg.det_type == 0:
        D[..., 0] = (cfg.dsd - cfg.dso) * c - t[None, :] * s
        D[..., 1] = (cfg.dsd - cfg.dso) * s + t[None, :] * c
    else:
        beta = t / cfg.dsd
        D[..., 0] = S[0] + cfg.dsd * np.cos(th + beta)[None, :]
        D[..., 1] = S[1] + cfg.dsd * np.sin(th + beta)[None, :]
    D[..., 2] = v[:, None]
    return S, D


def analytic_sinogram(cfg: Config, ellipses: list[Ellipse]) -> np.ndarray:
    """Exact line integrals, shape (nviews, nv, nu) fp64 (mm * mm^-1 = dimensionless)."""
    out = np.zeros((cfg.nviews, cfg.nv, cfg.nu))
    for k in range(cfg.nviews):
        S, D = ray_endpoints(cfg, k)
        d = D - S
        d /= np.linalg.norm(d, axis=-1, keepdims=True)
        acc = np.zeros(d.shape[:-1])
        for e in ellipses:
            cp, sp = math.cos(e.phi), math.sin(e.phi)
            inv_c = 0.0 if math.isinf(e.c) else 1.0 / e.c
            # rotate by -phi about z, scale by the semi-axes: ellipsoid -> unit sphere
            px = ((S[0] - e.x) * cp + (S[1] - e.y) * sp) / e.a
            py = (-(S[0] - e.x) * sp + (S[1] - e.y) * cp) / e.b
            pz = (S[2] - e.z) * inv_c
            ux = (d[..., 0] * cp + d[..., 1] * sp) / e.a
            uy = (-d[..., 0] * sp + d[..., 1] * cp) / e.b
            uz = d[..., 2] * inv_c
            uu = ux * ux + uy * uy + uz * uz
            pu = px * ux + py * uy + pz * uz
            pp = px * px + py * py + pz * pz
            disc = pu * pu - uu * (pp - 1.0)
            acc += e.dmu * 2.0 * np.sqrt(np.maximum(disc, 0.0)) / uu
        out[k] = acc
    return out


def add_poisson_noise(cfg: Config, sino: np.ndarray, slice_index: int = 0) -> np.ndarray:
    """BASELINE.json noise model: N~Poisson(I0 e^-y), y' = -ln(max(N,1)/I0)."""
    rng = _rng(cfg, slice_index, 1)
    counts = rng.poisson(cfg.I0 * np.exp(-sino)).astype(np.float64)
    return -np.log(np.maximum(counts, 1.0) / cfg.I0)


def rasterize(cfg: Config, ellipses: list[Ellipse], supersample: int = 2) -> np.ndarray:
    """Area-sampled raster (nz, ny, nx) fp64: mean of supersample^2 (2D) point samples per
    pixel; in 3D the z direction is point-sampled at the voxel centre."""
    ss = supersample
    sub = (np.arange(ss) + 0.5) / ss
    xs = (cfg.cx - cfg.nx * cfg.dx / 2.0) + (np.arange(cfg.nx)[:, None] + sub[None, :]).ravel() * cfg.dx
    ys = (cfg.cy - cfg.ny * cfg.dy / 2.0) + (np.arange(cfg.ny)[:, None] + sub[None, :]).ravel() * cfg.dy
    if cfg.ndim == 3:
        zs = (cfg.cz - cfg.nz * cfg.dz / 2.0) + (np.arange(cfg.nz) + 0.5) * cfg.dz
    else:
        zs = np.array([0.0])
    img = np.zeros((len(zs), cfg.ny, cfg.nx))
    for e in ellipses:
        cp, sp = math.cos(e.phi), math.sin(e.phi)
        rmax = max(e.a, e.b)
        ix = np.nonzero(np.abs(xs - e.x) <= rmax)[0]
        iy = np.nonzero(np.abs(ys - e.y) <= rmax)[0]
        if len(ix) == 0 or len(iy) == 0:
            continue
        x0, x1 = ix[0] // ss * ss, (ix[-1] // ss + 1) * ss
        y0, y1 = iy[0] // ss * ss, (iy[-1] // ss + 1) * ss
        X = xs[x0:x1][None, :] - e.x
        Y = ys[y0:y1][:, None] - e.y
        q = ((X * cp + Y * sp) / e.a) ** 2 + ((-X * sp + Y * cp) / e.b) ** 2
        for kz, z in enumerate(zs):
            qz = 0.0 if math.isinf(e.c) else ((z - e.z) / e.c) ** 2
            if qz >= 1.0:
                continue
            inside = (q + qz <= 1.0).astype(np.float64)
            cov = inside.reshape((y1 - y0) // ss, ss, (x1 - x0) // ss, ss).mean(axis=(1, 3))
            img[kz, y0 // ss:y1 // ss, x0 // ss:x1 // ss] += e.dmu * cov
    return img


def make_case(cfg: Config, slices=None, noisy: bool = True, raster: bool = True,
              supersample: int = 2):
    """Inputs of one workload as fp32 arrays in the ABI layouts.

    Returns dict(sino=[batch,nviews,nu] | [nviews,nv,nu], truth=[batch,ny,nx] | [nz,ny,nx]).
    `slices` selects a subset of the batch (2D only); default all of cfg.batch.
    """
    if cfg.ndim == 3:
        ell = make_phantom(cfg, 0)
        s = analytic_sinogram(cfg, ell)
        if noisy:
            s = add_poisson_noise(cfg, s, 0)
        out = {"sino": s.astype(np.float32)}
        if raster:
            out["truth"] = rasterize(cfg, ell, supersample).astype(np.float32)
        return out
    if slices is None:
        slices = range(cfg.batch)
    sinos, truths = [], []
    for sl in slices:
        ell = make_phantom(cfg, sl)
        s = analytic_sinogram(cfg, ell)[:, 0, :]
        if noisy:
            s = add_poisson_noise(cfg, s, sl)
        sinos.append(s.astype(np.float32))
        if raster:
            truths.append(rasterize(cfg, ell, supersample)[0].astype(np.float32))
    out = {"sino": np.stack(sinos)}
    if raster:
        out["truth"] = np.stack(truths)
    return out
