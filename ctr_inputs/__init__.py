"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This package holds NONE of the reconstruction method's arithmetic (no Siddon
traversal, no CGLS, no TV stencil): it only describes scanner geometries
(BASELINE.json configs c1..c5), draws seeded ellipse / ellipsoid phantoms,
evaluates their ANALYTIC line integrals (the "scanner simulator"), adds the
Poisson noise BASELINE.json prescribes and rasterises ground-truth images.
Neither `oracle/` nor `paper_1009_2288_b200/` is imported from here.
"""
from .configs import CONFIGS, Config, get_config, scaled_config
from .phantoms import (
    Ellipse,
    make_phantom,
    analytic_sinogram,
    add_poisson_noise,
    rasterize,
    make_case,
    ray_endpoints,
)

__all__ = [
    "CONFIGS", "Config", "get_config", "scaled_config", "Ellipse", "make_phantom",
    "analytic_sinogram", "add_poisson_noise", "rasterize", "make_case", "ray_endpoints",
]
