"""Closed-form helix truth used by the oracle pins (independent of oracle/ and of the CUDA path).

Conventions of the generator (paper_1910_12214_b200/datagen/tpcgen.cpp): a track starts at (0, 0, vz)
with global direction azimuth phi0; after turning angle psi its direction is phi0 - h*psi, its
distance from the beam line 2R sin(psi/2), z = vz + R psi sinh(eta); R = pT / (0.00299792458 Bz).
"""
import math

import numpy as np

KAPPA = 0.00299792458


def sector_alpha(sector: int) -> float:
    return ((sector % 18) + 0.5) * math.radians(20.0)


def truth_state_at_row(pt, phi0, eta, vz, h, bz, sector, x_row, n_sectors=36):
    """Local helix state (y, z, sin phi, dz/ds, q/pT) of the first crossing (psi in [0, pi)) of plane x_row.

    Returns None if the helix does not cross going outward.  q/pT follows d(sin phi)/dx = (q/pT) * KAPPA*Bz.
    """
    Rh = pt / (KAPPA * abs(bz))
    alpha = sector_alpha(sector) if n_sectors == 36 else math.radians(10.0)
    delta = phi0 - alpha
    v = math.sin(delta) - h * x_row / Rh
    if abs(v) >= 1:
        return None
    theta = math.asin(v)
    psi = h * (delta - theta)
    psi -= 2 * math.pi * math.floor(psi / (2 * math.pi))
    y = -h * Rh * (math.cos(delta) - math.cos(theta))
    tanl = math.sinh(eta)
    z = vz + Rh * psi * tanl
    q = -h / pt * (1.0 if bz >= 0 else -1.0)
    return np.array([y, z, v, tanl, q])


def helix_step_closed_form(state, dx, bz, longdouble=False):
    """Exact transport of (x, y, z, s, t, q) by dx along x in a uniform field (asin form).

    ``longdouble`` evaluates in x87 extended precision (the (c0 - c1)/k form cancels badly at small k*dx;
    the finite-difference Jacobian pin needs the extra digits).
    """
    f = np.longdouble if longdouble else np.float64
    x, y, z, s, t, q = (f(v) for v in state)
    dx = f(dx)
    k = q * f(KAPPA) * f(bz)
    s1 = s + dx * k
    c0, c1 = np.sqrt(1 - s * s), np.sqrt(1 - s1 * s1)
    if abs(k) < 1e-14:
        y1 = y + dx * s / c0
        dS = dx / c0
    else:
        y1 = y + (c0 - c1) / k
        dS = (np.arcsin(s1) - np.arcsin(s)) / k
    return np.array([x + dx, y1, z + t * dS, s1, t, q], dtype=f)


def tri(i, j):
    return i * (i + 1) // 2 + j if i >= j else j * (j + 1) // 2 + i


def cov_to_full(c15):
    C = np.zeros((5, 5))
    for i in range(5):
        for j in range(5):
            C[i, j] = c15[tri(i, j)]
    return C


def full_to_cov(C):
    return np.array([C[i, j] for i in range(5) for j in range(i + 1)])
