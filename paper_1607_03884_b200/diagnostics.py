"""Reported diagnostics of the path, computed from the product's own outputs (never from oracle/).

* divergence measure D of PAPER.md Eq. 3 (L190): per group of 32 consecutive IVPs (one warp of the paper's
  thread-per-IVP mapping), D = 1 - sum_i d_i / (32 max_i d_i), with d_i the number of internal integration steps the
  integrator took for IVP i (`chem_stats.nstep`).  The paper reports the distribution of D over the warps (Fig. 5,
  L192-L194); `divergence_summary` gives the same as a histogram over [0, 1].
* error metric E_i of Eq. 1 (L114-L116) and its maximum |E| of Eq. 2 (L118-L119), implemented as printed: a plain
  2-norm of (y - yhat) / (atol + yhat * rtol), yhat the "true" solution (reading "Error metric").
"""
from __future__ import annotations

import numpy as np


def divergence(d: np.ndarray) -> np.ndarray:
    """Eq. 3 for every complete group of 32 consecutive entries of d (a ragged tail is dropped, as in the paper's
    262,144 = 8192 x 32 IVPs).  A group whose maximum is 0 has D = 0."""
    d = np.asarray(d, dtype=np.int64)
    w = d.size // 32
    g = d[: w * 32].reshape(w, 32)
    mx = g.max(axis=1)
    out = np.zeros(w, dtype=np.float64)
    nz = mx > 0
    out[nz] = 1.0 - g[nz].sum(axis=1) / (32.0 * mx[nz])
    return out


def divergence_summary(d: np.ndarray, bins: int = 10) -> dict:
    """mean / median / 90th percentile of D and the share of warps per bin of width 1/bins (Fig. 5's histogram)."""
    D = divergence(d)
    if D.size == 0:
        return {"warps": 0, "mean": None, "p50": None, "p90": None, "hist": []}
    hist, _ = np.histogram(D, bins=bins, range=(0.0, 1.0))
    return {"warps": int(D.size), "mean": float(D.mean()), "p50": float(np.percentile(D, 50)),
            "p90": float(np.percentile(D, 90)), "hist": [round(float(h) / D.size, 4) for h in hist]}


def error_metric(y: np.ndarray, y_true: np.ndarray, rtol: float, atol: float):
    """Eq. 1 per IVP and Eq. 2 (their maximum).  Returns (|E|, E_i)."""
    y = np.asarray(y, dtype=np.float64)
    y_true = np.asarray(y_true, dtype=np.float64)
    E = np.sqrt((((y - y_true) / (atol + y_true * rtol)) ** 2).sum(axis=1))
    return (float(E.max()) if E.size else 0.0), E
