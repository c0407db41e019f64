"""Product-side diagnostics (paper_1607_03884_b200/diagnostics.py) against hand-computed values of PAPER.md Eq. 1-3."""
import numpy as np

from paper_1607_03884_b200 import diagnostics


def test_divergence_eq3_by_hand():
    # identical step counts -> D = 0; one thread with many steps -> D -> 1
    d = np.concatenate([np.full(32, 7), np.r_[np.full(31, 1), 100], np.arange(1, 33)])
    D = diagnostics.divergence(d)
    assert D.shape == (3,)
    assert D[0] == 0.0
    assert np.isclose(D[1], 1.0 - (31 + 100) / (32 * 100))
    assert np.isclose(D[2], 1.0 - (32 * 33 / 2) / (32 * 32))
    # ragged tail dropped; all-zero group has D = 0
    assert diagnostics.divergence(np.zeros(40, dtype=int)).tolist() == [0.0]
    assert diagnostics.divergence(np.arange(31)).size == 0


def test_divergence_summary_histogram():
    d = np.concatenate([np.full(32, 3)] * 3 + [np.r_[np.full(31, 1), 100]])
    s = diagnostics.divergence_summary(d, bins=10)
    assert s["warps"] == 4 and s["hist"][0] == 0.75 and s["hist"][9] == 0.25
    assert np.isclose(s["mean"], 0.25 * (1.0 - 131 / 3200))
    assert diagnostics.divergence_summary(np.arange(5))["warps"] == 0


def test_error_metric_eq1_eq2_by_hand():
    # Eq. 1 as printed: plain 2-norm of (y - yhat) / (atol + yhat rtol); Eq. 2: the maximum over the conditions
    yhat = np.array([[1000.0, 0.5], [2000.0, -0.25]])
    y = yhat + np.array([[1e-3, 1e-7], [0.0, 2e-7]])
    rtol, atol = 1e-6, 1e-10
    E0 = np.hypot(1e-3 / (atol + 1000.0 * rtol), 1e-7 / (atol + 0.5 * rtol))
    E1 = abs(2e-7 / (atol - 0.25 * rtol))        # yhat enters without modulus, as printed
    Emax, E = diagnostics.error_metric(y, yhat, rtol, atol)
    assert np.allclose(E, [E0, E1], rtol=1e-9) and np.isclose(Emax, max(E0, E1), rtol=1e-9)
