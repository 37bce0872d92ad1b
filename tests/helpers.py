"""Shared test helpers (no method arithmetic beyond norms and closed-form reference functions)."""
import math
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def golden(name):
    with open(os.path.join(ROOT, "tests", "golden", "paper_values.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            parts = line.split()
            if parts[0] == name:
                return float(parts[1])
    raise KeyError(name)


def hh_metric(x, y):
    """PAPER.md:246 Eq. 18."""
    return math.sqrt(((x - y) ** 2).sum() / (np.abs(x) * np.abs(y)).sum())


def rel_linf(a, b):
    return float(np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)).max()
                 / max(np.abs(np.asarray(b, dtype=np.float64)).max(), 1e-300))


def grid(nt, nphi):
    dth = math.pi / (nt + 1)
    dph = 2.0 * math.pi / nphi
    th = (np.arange(nt + 2) * dth)[:, None]
    ph = (np.arange(nphi) * dph)[None, :]
    return th, ph, dth, dph


def cell_areas(nt, nphi):
    """Quadrature weights under which the scheme conserves flux: sin(theta_j) dth dph, caps 2pi(1-cos(dth/2))."""
    th, ph, dth, dph = grid(nt, nphi)
    dA = np.sin(th) * dth * dph * np.ones((1, nphi))
    apole = 2.0 * math.pi * (1.0 - math.cos(dth / 2.0))
    dA[0, :] = apole / nphi      # the cap is one cell stored replicated over nphi columns
    dA[-1, :] = apole / nphi
    return dA


def soccer_ball(th, ph):
    """Eq. 19 spatial part: Y_6^0 + sqrt(14/11) Y_6^5 (real tesseral harmonics), scaled to max 1."""
    from scipy.special import sph_harm_y
    u = sph_harm_y(6, 0, th, ph).real + math.sqrt(14.0 / 11.0) * math.sqrt(2.0) * sph_harm_y(6, 5, th, ph).real
    return u / np.abs(u).max()
