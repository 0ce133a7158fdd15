"""The five workloads of BASELINE.json (`configs[0..4]` = c1..c5) as plain data.

Geometry fields carry the names of `ctr_geometry` (include/ctr.h); parameter
fields those of `ctr_params`.  Readings S13/S14 of SURVEY.md section 8(c) fix
what the paper leaves open (n_gd = 5, Armijo constants).
"""
from __future__ import annotations

import dataclasses
import math
import struct
from dataclasses import dataclass, field


def _f32(x: float) -> float:
    return struct.unpack("f", struct.pack("f", x))[0]


@dataclass(frozen=True)
class Config:
    name: str
    index: int                      # 1..5, enters the seed
    # --- geometry (ctr_geometry) ---
    ndim: int
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    nviews: int
    nu: int
    nv: int
    du: float
    dv: float
    dso: float
    dsd: float
    batch: int = 1
    cx: float = 0.0
    cy: float = 0.0
    cz: float = 0.0
    theta0: float = 0.0
    u_off: float = 0.0
    v_off: float = 0.0
    det_type: int = 0               # 0 = FLAT (all configs)
    # --- data ---
    I0: float = 1e4
    phantom: str = "c1"
    # --- ctr_params ---
    n_outer: int = 10
    n_cgls: int = 10
    n_gd: int = 5
    lam: float = 0.02
    sigma_quantile: float = 0.90
    eps: float = 1e-4
    armijo_t0: float = 1e-3
    armijo_rho: float = 0.5
    armijo_c: float = 0.5
    armijo_max: int = 16
    weights_mode: int = 0
    positivity: int = 1

    def __post_init__(self):
        # The C ABI carries every geometry / parameter scalar as fp32; the workload IS those fp32
        # values, so store each float field as the double of its fp32 rounding.
        for fld in dataclasses.fields(self):
            val = getattr(self, fld.name)
            if isinstance(val, float):
                object.__setattr__(self, fld.name, _f32(val))

    @property
    def dtheta(self) -> float:
        return _f32(2.0 * math.pi / self.nviews)

    @property
    def img_shape(self):
        if self.ndim == 3:
            return (self.nz, self.ny, self.nx)
        return (self.batch, self.ny, self.nx)

    @property
    def sino_shape(self):
        if self.ndim == 3:
            return (self.nviews, self.nv, self.nu)
        return (self.batch, self.nviews, self.nu)

    @property
    def n_rays(self) -> int:
        return self.nviews * self.nu * self.nv * self.batch

    @property
    def n_pix(self) -> int:
        return self.nx * self.ny * self.nz * self.batch

    def geometry_dict(self) -> dict:
        keys = ["ndim", "nx", "ny", "nz", "dx", "dy", "dz", "cx", "cy", "cz", "nviews",
                "theta0", "nu", "nv", "du", "dv", "u_off", "v_off", "dso", "dsd",
                "det_type", "batch"]
        d = {k: getattr(self, k) for k in keys}
        d["dtheta"] = self.dtheta
        return d

    def params_dict(self) -> dict:
        return dict(n_outer=self.n_outer, n_cgls=self.n_cgls, n_gd=self.n_gd,
                    lam=self.lam, sigma_quantile=self.sigma_quantile, eps=self.eps,
                    armijo_t0=self.armijo_t0, armijo_rho=self.armijo_rho,
                    armijo_c=self.armijo_c, armijo_max=self.armijo_max,
                    weights_mode=self.weights_mode, positivity=self.positivity)


CONFIGS = {
    # configs[0]: 64x64 @1.5 mm, 30 views x 96 bins @1.6 mm, I0=1e4, lambda=0.02, 10x10
    "c1": Config(name="c1", index=1, ndim=2, nx=64, ny=64, nz=1, dx=1.5, dy=1.5, dz=1.0,
                 nviews=30, nu=96, nv=1, du=1.6, dv=1.0, dso=541.0, dsd=949.0,
                 I0=1e4, phantom="c1", n_outer=10, n_cgls=10, lam=0.02),
    # configs[1]: 256x256 @1 mm, 40 views x 368 bins @1.2 mm, I0=5e3, lambda=0.02, 20x10
    "c2": Config(name="c2", index=2, ndim=2, nx=256, ny=256, nz=1, dx=1.0, dy=1.0, dz=1.0,
                 nviews=40, nu=368, nv=1, du=1.2, dv=1.0, dso=541.0, dsd=949.0,
                 I0=5e3, phantom="chest", n_outer=20, n_cgls=10, lam=0.02),
    # configs[2]: 512x512 @0.8 mm, 60 views x 888 bins @1.0 mm, I0=1e3, lambda=0.01, 30x15
    "c3": Config(name="c3", index=3, ndim=2, nx=512, ny=512, nz=1, dx=0.8, dy=0.8, dz=1.0,
                 nviews=60, nu=888, nv=1, du=1.0, dv=1.0, dso=541.0, dsd=949.0,
                 I0=1e3, phantom="catphan", n_outer=30, n_cgls=15, lam=0.01),
    # configs[3]: 64 slices of the c3 geometry, chest-like x1.6, I0=2e3, lambda=0.015, 30x15
    "c4": Config(name="c4", index=4, ndim=2, nx=512, ny=512, nz=1, dx=0.8, dy=0.8, dz=1.0,
                 nviews=60, nu=888, nv=1, du=1.0, dv=1.0, dso=541.0, dsd=949.0, batch=64,
                 I0=2e3, phantom="chest1.6", n_outer=30, n_cgls=15, lam=0.015),
    # configs[4]: cone beam 512x512x128 @0.8 mm, 60 views, 512(u) x 384(v) @0.78 mm,
    # dso 1000, dsd 1500, I0=5e3, lambda=0.01, 20x10
    "c5": Config(name="c5", index=5, ndim=3, nx=512, ny=512, nz=128, dx=0.8, dy=0.8, dz=0.8,
                 nviews=60, nu=512, nv=384, du=0.78, dv=0.78, dso=1000.0, dsd=1500.0,
                 I0=5e3, phantom="chest3d", n_outer=20, n_cgls=10, lam=0.01),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]


def scaled_config(name: str, **overrides) -> Config:
    """A config with some fields replaced (smaller batch, fewer iterations, ...)."""
    return dataclasses.replace(CONFIGS[name], **overrides)
