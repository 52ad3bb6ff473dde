"""Error metrics of BASELINE.json north_star (readings Q17, Q18 in DESIGN.md)."""
from __future__ import annotations

import numpy as np


def field_errors(H_test, H_ref):
    """Returns (max_c rel-L2, max-abs rel): e_c = ||H_c - Href_c||_2 / (sqrt(n) max|Href|),
    and max|H - Href| / max|Href|."""
    a = np.asarray(H_test, dtype=np.float64).reshape(-1, 3)
    b = np.asarray(H_ref, dtype=np.float64).reshape(-1, 3)
    scale = np.max(np.abs(b))
    if scale == 0.0:
        scale = 1.0
    d = a - b
    l2 = np.sqrt(np.mean(d * d, axis=0)) / scale
    return float(np.max(l2)), float(np.max(np.abs(d)) / scale)


def traj_error(m_test, m_ref):
    """max over cells and components of |m_test - m_ref|."""
    return float(np.max(np.abs(np.asarray(m_test, dtype=np.float64) - np.asarray(m_ref))))
