"""Scalar inputs of the step that the paper gives in closed form: critical stretch s_c
(Eqs. 1.26-1.29) and the wave-speed time-step bound (Eq. 2.13).

TEST INFRASTRUCTURE (same rule as the rest of oracle/).  These scalars are INPUTS of the
library (pd_material.s_c, pd_material.dt): GPU/oracle parity never depends on them.  The
literals the workload generators carry were written by oracle/derive_scalars.py from these
functions.
"""
from __future__ import annotations

import math

MODE_3D, MODE_PLANE_STRESS, MODE_PLANE_STRAIN = 0, 1, 2


def moduli(E: float, nu: float):
    """kappa, mu, lambda."""
    kappa = E / (3.0 * (1.0 - 2.0 * nu))
    mu = E / (2.0 * (1.0 + nu))
    lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu))
    return kappa, mu, lam


def beta_constants(mode: int, delta: float, variant: str = "printed"):
    """beta, beta' for w = 1.  'printed': Eq. 1.27 / Eq. 1.29
     exactly as printed.  'integrated': what direct integration of
    Eqs. 1.22/1.25 gives (3D beta' = 5 delta/24 without the pi; reading C-9)."""
    if mode == MODE_3D:
        beta = 125.0 * delta / 1848.0
        bprime = 5.0 * delta / (24.0 * math.pi) if variant == "printed" else 5.0 * delta / 24.0
    else:
        beta = 1087.0 * delta / (1250.0 * math.pi ** 2)
        bprime = 4.0 * delta / (5.0 * math.pi)
    return beta, bprime


def critical_stretch(mode: int, E: float, nu: float, G0: float, delta: float,
                     variant: str = "printed") -> float:
    """s_c of Eq. 1.26 (3D) or Eq. 1.28 (2D)."""
    kappa, mu, _ = moduli(E, nu)
    beta, bprime = beta_constants(mode, delta, variant)
    if mode == MODE_3D:
        den = (9.0 * kappa - 15.0 * mu) * beta + 15.0 * mu * bprime
    else:
        if mode == MODE_PLANE_STRESS:
            A = 2.0 * (1.0 - 2.0 * nu) / (1.0 - nu)
            kp = kappa + (mu / 9.0) * ((1.0 + nu) / (1.0 - 2.0 * nu)) ** 2
        else:
            A = 2.0
            kp = kappa + mu / 9.0
        den = A * A * (kp - 8.0 * mu / 9.0) * beta + 8.0 * mu * bprime
    if den <= 0.0:
        raise ValueError("non-positive radicand in Eq. 1.26/1.28")
    return math.sqrt(G0 / den)


def wave_speed_bound(E: float, nu: float, rho: float, delta: float) -> float:
    """delta / c', c' = sqrt((lambda + 2 mu)/rho)  (Eq. 2.13)."""
    _, mu, lam = moduli(E, nu)
    return delta / math.sqrt((lam + 2.0 * mu) / rho)
