"""Image-quality metrics of the paper's evaluation section (NEXT-3; harness side, numpy only, no arithmetic of
the reconstruction method): relative error Eq. (12), edge cross-correlation Eq. (13), SNR Eq. (14)."""
from __future__ import annotations

import numpy as np


def relative_error(f, f_true) -> float:
    """Eq. (12), as printed: e = ||f - f*||_2^2 / ||f*||_2^2 (squared norms)."""
    f, f_true = np.asarray(f, np.float64), np.asarray(f_true, np.float64)
    return float(((f - f_true) ** 2).sum() / (f_true ** 2).sum())


def sobel_edges(img, threshold_fraction: float = 0.1) -> np.ndarray:
    """Binary edge map b of Eq. (13): Sobel gradient magnitude (Kanopoulos et al. 1988) above
    threshold_fraction x its maximum. The paper does not print its threshold: it is a parameter here."""
    a = np.pad(np.asarray(img, np.float64), 1, mode="edge")
    gx = (a[:-2, 2:] + 2 * a[1:-1, 2:] + a[2:, 2:]) - (a[:-2, :-2] + 2 * a[1:-1, :-2] + a[2:, :-2])
    gy = (a[2:, :-2] + 2 * a[2:, 1:-1] + a[2:, 2:]) - (a[:-2, :-2] + 2 * a[:-2, 1:-1] + a[:-2, 2:])
    mag = np.hypot(gx, gy)
    top = mag.max()
    return (mag > threshold_fraction * top) if top > 0 else np.zeros(mag.shape, bool)


def edge_cross_correlation(f, f_true, threshold_fraction: float = 0.1) -> float:
    """Eq. (13): correlation coefficient of the two binary edge maps."""
    b = sobel_edges(f, threshold_fraction).astype(np.float64).ravel()
    bt = sobel_edges(f_true, threshold_fraction).astype(np.float64).ravel()
    b, bt = b - b.mean(), bt - bt.mean()
    den = np.sqrt((b * b).sum() * (bt * bt).sum())
    return float((b * bt).sum() / den) if den > 0 else 0.0


def snr_db(img, roi) -> float:
    """Eq. (14): 10 log10( E(P)^2 / E([P - E(P)]^2) ) over the pixels P selected by `roi`
    (a boolean mask or a tuple of slices)."""
    p = np.asarray(img, np.float64)[roi].ravel()
    m = p.mean()
    var = ((p - m) ** 2).mean()
    return float(10.0 * np.log10(m * m / var)) if var > 0 else float("inf")
