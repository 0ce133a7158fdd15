"""Eq. (12)-(14) of the paper (NEXT-3 harness) against hand-computable cases."""
import numpy as np
import pytest

from ctr_inputs import metrics


def test_relative_error_eq12():
    f = np.arange(12.0).reshape(3, 4) + 1
    assert metrics.relative_error(f, f) == 0.0
    assert metrics.relative_error(2 * f, f) == pytest.approx(1.0)            # squared norms, as printed
    assert metrics.relative_error(1.1 * f, f) == pytest.approx(0.01)


def test_snr_eq14():
    roi = (slice(0, 2), slice(0, 2))
    img = np.array([[9.0, 11.0, 100.0], [11.0, 9.0, -5.0]])
    # ROI values 9, 11, 11, 9: mean 10, variance 1 -> 10 log10(100) = 20 dB
    assert metrics.snr_db(img, roi) == pytest.approx(20.0)
    assert metrics.snr_db(np.ones((4, 4)), np.ones((4, 4), bool)) == float("inf")


def test_edge_cross_correlation_eq13():
    a = np.zeros((32, 32)); a[:, 16:] = 1.0                      # one vertical edge
    b = np.zeros((32, 32)); b[16:, :] = 1.0                      # one horizontal edge
    assert metrics.edge_cross_correlation(a, a) == pytest.approx(1.0)
    assert metrics.edge_cross_correlation(a, 3.0 * a + 2.0) == pytest.approx(1.0)   # edges, not intensities
    assert abs(metrics.edge_cross_correlation(a, b)) < 0.2
    e = metrics.sobel_edges(a)
    assert e[:, 15:17].all() and not e[:, :14].any() and not e[:, 18:].any()
    assert metrics.edge_cross_correlation(np.ones((8, 8)), a[:8, :8]) == 0.0
