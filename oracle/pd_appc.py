"""Second, independent formulation of the force: the paper's LOOP scheme (App. C,
PAPER.md:888-937) and its explicit solver body (App. B) in numpy.

TEST INFRASTRUCTURE (same rule as pd_oracle.c: only tests/, smoke() and bench.py's CPU legs).
It exists so that the gather oracle (pd_oracle.c) can be cross-checked against a code with a
different data structure (one entry per UNDIRECTED bond, pair scatter instead of gather) and
a different arithmetic arrangement.  It shares nothing with pd_oracle.c.

Deviations from the App. C listing, all listed in DESIGN.md:
  * extension is the LINEARIZED one, e = M . (u_j - u_i) (reading C-1; the listing computes
    the geometric ||xi+eta|| - ||xi||);
  * the three typos are fixed per Eq. 2.2 (reading C-12): `Theta(index2)=Theta(index1)+...`
    accumulates into Theta(index2); `DE2=E(i)/m(index1)` uses m(index2); PDF has dim*Nn
    entries.  The second division of Theta by m (PAPER.md:920 then :925) is kept: Eq. 2.2.
  * PDF here is the nodal FORCE (x V_i V_j) exactly as in App. C; divide by V_i for the
    force density of Eq. 2.1.
"""
from __future__ import annotations

import numpy as np


def bond_list(coords: np.ndarray, horizon: float):
    """BondList(Nb,2) with i<j, Xi (bond vectors) and xi (lengths) -- App. C's inputs.
    O(N^2) broadcasting: small models only."""
    x = np.asarray(coords, dtype=np.float64)
    d = x[None, :, :] - x[:, None, :]
    r2 = np.zeros(d.shape[:2])
    for k in range(x.shape[1]):
        r2 = r2 + d[:, :, k] * d[:, :, k]
    i, j = np.nonzero(np.triu(r2 <= horizon * horizon, k=1))
    Xi = x[j] - x[i]
    return np.stack([i, j], axis=1), Xi, np.sqrt(np.sum(Xi * Xi, axis=1))


def weighted_volume(n, bonds, xi, vol):
    """m of Eq. 1.9 by pair iteration (both directions of each stored pair contribute)."""
    m = np.zeros(n)
    np.add.at(m, bonds[:, 0], xi * xi * vol[bonds[:, 1]])
    np.add.at(m, bonds[:, 1], xi * xi * vol[bonds[:, 0]])
    return m


def pd_force(U, vol, bonds, m, xi, Xi, co_index, A, K, G, geometric=False):
    """PDForceComputLoop of App. C (vectorised over bonds; np.add.at plays the loop).
    U: (Nn, dim).  Returns PDF (Nn, dim) nodal forces and Theta.
    geometric=True keeps the extension exactly as the listing prints it."""
    n, dim = U.shape
    i1, i2 = bonds[:, 0], bonds[:, 1]
    M = Xi / xi[:, None]
    if geometric:
        Eta = Xi + (U[i2] - U[i1])
        E = np.sqrt(np.sum(Eta * Eta, axis=1)) - xi
    else:
        E = np.sum(M * (U[i2] - U[i1]), axis=1)      # linearized (Eq. 2.7)
    E = np.where(co_index == 0, 0.0, E)
    theta = np.zeros(n)
    np.add.at(theta, i1, A * xi * E * co_index * vol[i2])
    np.add.at(theta, i2, A * xi * E * co_index * vol[i1])   # PAPER.md:918 (typo fixed)
    theta = theta / m
    DT1, DT2 = theta[i1] / m[i1], theta[i2] / m[i2]
    DE1, DE2 = E / m[i1], E / m[i2]                          # PAPER.md:926 (typo fixed)
    FT = (K - G / 3.0) * (DT1 + DT2) * xi * co_index * vol[i1] * vol[i2]
    FE = G * (DE1 + DE2) * co_index * vol[i1] * vol[i2]
    PDF = np.zeros((n, dim))
    np.add.at(PDF, i1, ((FT + FE)[:, None]) * M)
    np.add.at(PDF, i2, -((FT + FE)[:, None]) * M)
    return PDF, theta


def run_explicit(coords, vol, horizon, A, K, G, rho_mass, dt, nsteps, u0, v0, clamp_mask,
                 s_c=0.0, co_index=None):
    """App. B solver body with the App. C force, free/clamped dofs only (no loads).
    clamp_mask: (Nn, dim) bool.  Returns U, VEL, co_index, list of (step, i, j) breaks."""
    coords = np.asarray(coords, dtype=np.float64)
    n, dim = coords.shape
    bonds, Xi, xi = bond_list(coords, horizon)
    m = weighted_volume(n, bonds, xi, vol)
    co = np.ones(len(bonds)) if co_index is None else np.asarray(co_index, dtype=np.float64).copy()
    U = np.array(u0, dtype=np.float64).reshape(n, dim).copy()
    VEL = np.array(v0, dtype=np.float64).reshape(n, dim).copy()
    U[clamp_mask] = 0.0
    VEL[clamp_mask] = 0.0
    Mass = rho_mass * vol[:, None]                            # lumped mass rho V_i
    breaks = []
    M = Xi / xi[:, None]
    for it in range(nsteps):
        PDF, _ = pd_force(U, vol, bonds, m, xi, Xi, co, A, K, G)
        ACC = PDF / Mass                                      # RF=EXF+PDF; ACC=RF./M
        VEL = VEL + ACC * dt
        VEL[clamp_mask] = 0.0
        U = np.where(clamp_mask, U, U + dt * VEL)
        if s_c > 0.0:
            s = np.sum(M * (U[bonds[:, 1]] - U[bonds[:, 0]]), axis=1) / xi
            newly = (co != 0) & (s >= s_c)
            for b in np.nonzero(newly)[0]:
                breaks.append((it, int(bonds[b, 0]), int(bonds[b, 1])))
            co[newly] = 0.0
    return U, VEL, co, breaks
