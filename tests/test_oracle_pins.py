"""Pins of the CPU oracle (oracle/pd_oracle.c) against what the paper and the mathematics fix.

None of these re-types the oracle's formulas: they are printed values, closed
forms, invariants, hand-computed tiny systems (tests/golden/paper_values.json), special cases
and brute force.  A dropped term, wrong sign/index or transposed operand in any oracle
function fails at least one of them (see DESIGN.md "Oracle pins" for the mapping).
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import pd_appc, scalars
from oracle.pd_oracle import (MODE_3D, MODE_PLANE_STRAIN, MODE_PLANE_STRESS, PDOracle, constants,
                              family)

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
MODES = [(3, MODE_3D), (2, MODE_PLANE_STRESS), (2, MODE_PLANE_STRAIN)]


def lattice(shape, dx=1.0):
    g = np.stack(np.meshgrid(*[np.arange(s) for s in shape], indexing="ij"), axis=-1)
    return (g.reshape(-1, len(shape)) + 0.5) * dx


def make(coords, dim, mode, horizon, E=72e9, nu=0.22, rho=2440.0, dt=1e-7, vol=None, **kw):
    coords = np.asarray(coords, float).reshape(-1, dim)
    vol = np.full(len(coords), 1.0) if vol is None else vol
    return PDOracle(coords, vol, horizon, dim=dim, mode=mode, E=E, nu=nu, rho=rho, dt=dt, **kw)


# ---- family ---------------------------------------------------------------------------------
def test_1058_bonds_paper():
    """10x10 nodes, m-ratio 3 -> 1058 bonds (inclusive horizon, reading C-11)."""
    rp, col = family(lattice((10, 10)), 3.0, "brute")
    assert rp[-1] == 2 * GOLD["bonds_10x10_mratio3"]["value"]
    rp2, col2 = family(lattice((10, 10)), 3.0, "cells")
    assert np.array_equal(rp, rp2) and np.array_equal(col, col2)


@pytest.mark.parametrize("shape,interior", [((9, 9), 28), ((7, 7, 7), 122)])
def test_interior_family_and_lattice_total(shape, interior):
    x = lattice(shape)
    rp, col = family(x, 3.015, "cells")
    centre = np.argmin(np.sum((x - x.mean(0)) ** 2, axis=1))
    assert rp[centre + 1] - rp[centre] == interior
    r = np.arange(-3, 4)
    offs = np.stack(np.meshgrid(*([r] * len(shape)), indexing="ij"), -1).reshape(-1, len(shape))
    offs = offs[(np.sum(offs ** 2, 1) > 0) & (np.sum(offs ** 2, 1) <= 9)]
    total = sum(int(np.prod([max(0, n - abs(o)) for n, o in zip(shape, off)])) for off in offs)
    assert rp[-1] == total


def test_config1_bond_total():
    """100x10 lattice -> Z = 24 076 directed bonds (offset-sum formula)."""
    rp, _ = family(lattice((100, 10)), 3.015)
    assert rp[-1] == 24076


@pytest.mark.parametrize("dim", [2, 3])
def test_brute_equals_cells_random_cloud(dim):
    rng = np.random.default_rng(5)
    x = rng.uniform(0, 10, size=(1500 if dim == 2 else 3000, dim))
    a = family(x, 1.3, "brute")
    b = family(x, 1.3, "cells")
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert a[0][-1] > 0
    # symmetric: (i,j) present <=> (j,i) present; rows ascending
    i = np.repeat(np.arange(len(x)), np.diff(a[0]))
    s1 = set(zip(i.tolist(), a[1].tolist()))
    assert s1 == {(q, p) for p, q in s1}
    for r in range(len(x)):
        row = a[1][a[0][r]:a[0][r + 1]]
        assert np.all(np.diff(row) > 0) and r not in row


def test_family_permutation_invariance():
    x = lattice((12, 7))
    perm = np.random.default_rng(1).permutation(len(x))
    rp, col = family(x, 3.015)
    rq, cq = family(x[perm], 3.015)
    i = np.repeat(np.arange(len(x)), np.diff(rp))
    iq = np.repeat(np.arange(len(x)), np.diff(rq))
    assert set(zip(i.tolist(), col.tolist())) == set(zip(perm[iq].tolist(), perm[cq].tolist()))


# ---- weighted volume ------------------------------------------------------------------------
def test_m_two_nodes_and_interior():
    o = make([[0, 0, 0], [0.3, 0.4, 0.0]], 3, MODE_3D, 1.0, vol=np.array([2.0, 5.0]))
    assert np.allclose(o.m, [0.25 * 5.0, 0.25 * 2.0], rtol=1e-15)
    assert np.allclose(o.fvol, [5.0, 2.0])
    for shape, dim, mode, key in [((9, 9), 2, MODE_PLANE_STRESS, "2d"), ((7, 7, 7), 3, MODE_3D, "3d")]:
        dx, V = 0.5, 0.125
        x = lattice(shape, dx)
        o = make(x, dim, mode, 3.015 * dx, vol=np.full(len(x), V))
        c = np.argmin(np.sum((x - x.mean(0)) ** 2, axis=1))
        assert o.m[c] == pytest.approx(GOLD["interior_m_over_dx2V"][key] * dx * dx * V, rel=1e-14)


# ---- constants ------------------------------------------------------------------------------
def test_constants_identities():
    for nu in (0.1, 0.22, 0.3, 1 / 3):
        E = 72e9
        A, K, G, kappa, mu = constants(MODE_PLANE_STRESS, E, nu)
        assert K == pytest.approx(kappa, rel=1e-13)          # Eq. 1.15 plane stress simplifies to kappa
        assert A == pytest.approx(2 * (1 - 2 * nu) / (1 - nu))
        A3, K3, G3, _, _ = constants(MODE_3D, E, nu)
        assert (A3, K3, G3) == (3.0, 3 * kappa, 15 * mu)
        A2, K2, G2, _, _ = constants(MODE_PLANE_STRAIN, E, nu)
        assert (A2, G2) == (2.0, 8 * mu) and K2 == pytest.approx(2 * kappa - 2 * mu / 3)
    A, _, _, _, _ = constants(MODE_PLANE_STRESS, 1.0, 1 / 3)
    assert A == pytest.approx(1.0)
    with pytest.raises(ValueError):
        constants(MODE_3D, 1.0, 0.5)


# ---- dilatation -----------------------------------------------------------------------------
@pytest.mark.parametrize("dim,mode", MODES)
def test_uniform_stretch_theta_and_energy(dim, mode):
    """u = eps x  =>  theta_i = A eps at EVERY node (m cancels, Eq. 1.6), and W_i equals the
    classical strain energy of that state (Eq. 1.20 with the mode constants)."""
    shape = (9, 8, 7) if dim == 3 else (12, 9)
    dx, eps, E, nu = 1e-3, 1e-4, 72e9, 0.22
    x = lattice(shape, dx)
    x = x + np.random.default_rng(0).uniform(-0.05 * dx, 0.05 * dx, x.shape)  # irregular on purpose
    o = make(x, dim, mode, 3.015 * dx, E=E, nu=nu, vol=np.full(len(x), dx ** dim))
    th = o.dilatation(eps * x).copy()
    assert np.allclose(th, o.A * eps, rtol=1e-12)
    W = o.energy_density(eps * x)
    kappa, mu = o.kappa, o.mu
    classical = {MODE_3D: 4.5 * kappa * eps ** 2, MODE_PLANE_STRAIN: (2 * kappa + 2 * mu / 3) * eps ** 2,
                 MODE_PLANE_STRESS: E * eps ** 2 / (1 - nu)}[mode]
    assert np.allclose(W, classical, rtol=1e-11)


@pytest.mark.parametrize("dim,mode", MODES)
def test_homogeneous_strain_interior_theta(dim, mode):
    """general homogeneous strain on an interior node of the unjittered lattice:
    theta = (A/d) tr(eps) (second moment of a symmetric family is isotropic)."""
    shape = (7, 7, 7) if dim == 3 else (9, 9)
    x = lattice(shape, 1.0)
    rng = np.random.default_rng(3)
    Hm = rng.standard_normal((dim, dim)) * 1e-4
    o = make(x, dim, mode, 3.015, vol=np.full(len(x), 1.0))
    th = o.dilatation(x @ Hm.T)
    c = np.argmin(np.sum((x - x.mean(0)) ** 2, axis=1))
    assert th[c] == pytest.approx(o.A / dim * np.trace(Hm), rel=1e-11)


# ---- force ----------------------------------------------------------------------------------
def _random_sym_mask(o, frac, seed):
    rng = np.random.default_rng(seed)
    i, j = o.bond_pairs()
    key = np.minimum(i, j) * o.n + np.maximum(i, j)
    uniq = np.unique(key)
    dead = set(uniq[rng.random(len(uniq)) < frac].tolist())
    o.rho[:] = np.array([0 if k in dead else 1 for k in key.tolist()], dtype=np.uint8)


@pytest.mark.parametrize("dim,mode", MODES)
def test_rigid_motion_zero_force_and_balance(dim, mode):
    shape = (8, 7, 6) if dim == 3 else (11, 9)
    dx = 1e-3
    x = lattice(shape, dx) + np.random.default_rng(1).uniform(-0.1 * dx, 0.1 * dx, (int(np.prod(shape)), dim))
    vol = np.random.default_rng(2).uniform(0.5, 1.5, len(x)) * dx ** dim     # non-uniform volumes
    o = make(x, dim, mode, 3.015 * dx, vol=vol)
    rng = np.random.default_rng(4)
    u = rng.standard_normal(x.shape) * 1e-6
    scale = np.max(np.abs(o.force_density(u)))
    assert scale > 0
    # rigid translation, infinitesimal rotation u = W x with W skew
    assert np.max(np.abs(o.force_density(np.ones_like(x) * 3e-6))) <= 1e-10 * scale
    Wm = rng.standard_normal((dim, dim)); Wm = (Wm - Wm.T) * 1e-3
    assert np.max(np.abs(o.force_density(x @ Wm.T))) <= 1e-9 * scale
    # momentum and angular momentum balance for any u and any SYMMETRIC mask
    _random_sym_mask(o, 0.15, 9)
    f = o.force_density(u).copy()
    F = f * vol[:, None]
    assert np.max(np.abs(F.sum(0))) <= 1e-10 * np.abs(F).sum()
    if dim == 2:
        tq = np.sum(x[:, 0] * F[:, 1] - x[:, 1] * F[:, 0])
    else:
        tq = np.abs(np.cross(x, F).sum(0)).max()
    assert abs(tq) <= 1e-10 * np.abs(F).sum() * np.abs(x).max()
    # linearity
    u2 = rng.standard_normal(x.shape) * 1e-6
    f2 = o.force_density(u2).copy()
    f12 = o.force_density(2.0 * u - 3.0 * u2)
    assert np.allclose(f12, 2.0 * f - 3.0 * f2, rtol=0, atol=1e-10 * scale)
    # energy: Pi = sum V W  equals  -1/2 sum u . V f   (Eq. 1.20 vs Eq. 2.1)
    W = o.energy_density(u)
    assert np.sum(vol * W) == pytest.approx(-0.5 * np.sum(u * F), rel=1e-10)


def test_two_node_hand_values():
    g = GOLD["two_node"]; assert "18*kappa" in g["F1_3d"]
    r, V, a, E, nu = 0.7, 0.3, 2e-4, 5.0, 0.2
    d = np.array([0.6, 0.0, 0.8]) * r                              # bond direction, |d| = r
    o = make([[0, 0, 0], d], 3, MODE_3D, 1.0, E=E, nu=nu, vol=np.full(2, V))
    u = np.array([[0, 0, 0], a * d / r])
    th = o.dilatation(u).copy()
    assert np.allclose(th, 3 * a / r, rtol=1e-14)
    F = o.force_density(u) * V
    assert np.allclose(F[0], 18 * o.kappa * a * V / r ** 2 * d / r, rtol=1e-13)
    assert np.allclose(F[1], -F[0], rtol=1e-15)
    o2 = make([[0, 0], d[[0, 2]]], 2, MODE_PLANE_STRAIN, 1.0, E=E, nu=nu, vol=np.full(2, V))
    u2 = np.array([[0, 0], a * d[[0, 2]] / r])
    assert np.allclose(o2.dilatation(u2), 2 * a / r, rtol=1e-14)
    F2 = o2.force_density(u2) * V
    assert np.allclose(F2[0], 8 * (3 * o2.kappa + o2.mu) * a * V / (3 * r ** 2) * d[[0, 2]] / r, rtol=1e-13)


def test_three_node_hand_values():
    g = GOLD["three_node"]
    # kappa = mu = 1  <=>  E = 9 kappa mu/(3 kappa + mu) = 9/4, nu = (3k-2mu)/(2(3k+mu)) = 1/8
    o = make([[0, 0, 0], [1, 0, 0], [2, 0, 0]], 3, MODE_3D, 2.0, E=2.25, nu=0.125, vol=np.ones(3))
    assert o.kappa == pytest.approx(1.0, rel=1e-15) and o.mu == pytest.approx(1.0, rel=1e-15)
    assert np.allclose(o.m, g["m"], rtol=1e-15)
    u = np.array([[0, 0, 0], [0.01, 0, 0], [0.03, 0, 0]])
    th = o.dilatation(u).copy()
    assert np.allclose(th, [float(Fraction(s)) for s in g["theta"]], rtol=1e-14)
    F = o.force_density(u)                                       # V = 1: force = density
    assert np.allclose(F[:, 0], [float(Fraction(s)) for s in g["F"]], rtol=1e-13)
    assert np.all(F[:, 1:] == 0.0)


# ---- integrator -----------------------------------------------------------------------------
def test_constant_force_closed_form():
    """Eq. 2.11 from rest under constant acceleration: U_n = (b/rho) dt^2 n(n+1)/2.
    Two nodes with the same body force move together, so no internal force arises."""
    b, rho, dt, n = 3.0e4, 2440.0, 1e-6, 37
    o = make([[0, 0], [1, 0]], 2, MODE_PLANE_STRESS, 1.5, rho=rho, dt=dt,
             flags=np.array([64, 64], np.uint8), value=np.array([[0, b], [0, b]]))
    o.step(n)
    assert np.allclose(o.u[:, 1], (b / rho) * dt * dt * n * (n + 1) / 2, rtol=1e-13)
    assert np.all(o.u[:, 0] == 0.0)
    assert np.allclose(o.v[:, 1], (b / rho) * dt * n, rtol=1e-13)


def test_ramp_clamp_prescribed():
    """g(t_n) = min(1, n dt/ramp): sum_{k<n} g_k closed form; clamp holds u=0,v=0;
    prescribed dof moves at vbar exactly (readings C-3, C-4, C-14)."""
    b, rho, dt, n, nr = 1.0e5, 1000.0, 1e-6, 30, 10
    x = [[0, 0], [1, 0], [5, 0], [6, 0]]
    flags = np.array([64, 64, 1 | 2, 8], np.uint8)
    value = np.array([[b, 0], [b, 0], [0, 0], [2.5, 0]])
    o = make(x, 2, MODE_PLANE_STRAIN, 1.5, rho=rho, dt=dt, ramp_time=nr * dt, flags=flags, value=value,
             u0=np.array([[0, 0], [0, 0], [7., 7.], [0, 0]]), v0=np.array([[0, 0], [0, 0], [1., 1.], [0, 0]]))
    o.step(n)
    gs = np.minimum(1.0, np.arange(n) / nr)
    v_expected = (b / rho) * dt * gs.sum()
    u_expected = (b / rho) * dt * dt * np.cumsum(gs).sum()
    assert np.allclose(o.v[:2, 0], v_expected, rtol=1e-12)
    assert np.allclose(o.u[:2, 0], u_expected, rtol=1e-12)
    assert np.all(o.u[2] == 0.0) and np.all(o.v[2] == 0.0)
    # node 3 is bonded to the clamped node 2; its x dof is driven, y dof free (but no y force)
    assert o.v[3, 0] == 2.5 and o.u[3, 0] == pytest.approx(2.5 * dt * n, rel=1e-13)


def test_modified_energy_invariant_config1():
    """Exact invariant of Eq. 2.11 for a fixed mask and no load:
    H~ = 1/2 sum rho V |v|^2 + Pi(u) + (dt/2) sum v . V f(u), conserved to roundoff, while the
    plain energy oscillates.  Run on config 1 at its dt = 0.8 x critical for 2000 steps."""
    from paper_2309_11273_b200 import workloads
    wl = workloads.cantilever2d()
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, u0=wl.u0)
    free = np.ones((wl.n, 2), bool)
    free[(wl.flags & 1) != 0, 0] = False
    free[(wl.flags & 2) != 0, 1] = False

    def H():
        f = o.force_density().copy()
        Pi = np.sum(wl.volumes * o.energy_density())
        ke = 0.5 * wl.rho * np.sum(wl.volumes[:, None] * o.v ** 2)
        cross = 0.5 * wl.dt * np.sum((o.v * f * wl.volumes[:, None])[free])
        return ke + Pi + cross, ke + Pi

    h0, e0 = H()
    hs, es = [h0], [e0]
    for _ in range(20):
        o.step(100)
        h, e = H(); hs.append(h); es.append(e)
    hs, es = np.array(hs), np.array(es)
    assert np.max(np.abs(hs - h0)) <= 1e-11 * abs(h0)
    assert np.max(np.abs(es - e0)) > 1e-6 * abs(e0)       # the plain energy is NOT the invariant
    assert np.all(np.isfinite(o.u)) and np.max(np.abs(o.u)) < 1e-4   # stable at this dt


# ---- failure / damage -----------------------------------------------------------------------
def test_single_bond_breaks_at_threshold():
    s_c = 1e-3
    for a, broken in [(s_c, True), (np.nextafter(s_c, 0), False), (-5 * s_c, False)]:
        o = make([[0, 0], [1, 0]], 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, u0=np.array([[0, 0], [a, 0.0]]))
        nb, _ = o.break_bonds()
        assert (nb == 2) == broken and bool(o.rho.sum() == 0) == broken
        assert np.allclose(o.damage(), 1.0 if broken else 0.0)
    # no-fail end keeps the bond
    o = make([[0, 0], [1, 0]], 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, u0=np.array([[0, 0], [2 * s_c, 0.0]]),
             flags=np.array([0, 128], np.uint8))
    assert o.break_bonds()[0] == 0


def test_near_threshold_counter():
    """the oracle's near-threshold counter (north star: bonds within 1e-9 relative of s_c at the step they
    break "are counted and reported"): a bond at s_c (1 +- 5e-10) is counted (in both directions), one at
    s_c (1 +- 1e-8) is not; the counter is independent of whether the bond breaks; step() accumulates it"""
    s_c = 1e-3
    for rel, near in [(+5e-10, 2), (-5e-10, 2), (+1e-8, 0), (-1e-8, 0), (0.0, 2)]:
        a = s_c * (1.0 + rel)
        o = make([[0, 0], [1, 0]], 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, u0=np.array([[0, 0], [a, 0.0]]))
        nb, nn = o.break_bonds(near_tol=1e-9)
        assert nn == near, (rel, nn)
        assert nb == (2 if rel >= 0 else 0)
    # through the time stepper: both dofs of both nodes carry a prescribed velocity 0, so u^1 = u^0
    a = s_c * (1.0 - 5e-10)
    o = make([[0, 0], [1, 0]], 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, u0=np.array([[0, 0], [a, 0.0]]),
             flags=np.array([24, 24], np.uint8), value=np.zeros((2, 2)), dt=1e-9)
    assert o.step(3) == 0 and o.near_total == 6   # 2 directed bonds x 3 steps, never breaking


def test_damage_half_family_and_precut_band():
    x = lattice((9, 9))
    o = make(x, 2, MODE_PLANE_STRESS, 3.015)
    c = int(np.argmin(np.sum((x - x.mean(0)) ** 2, axis=1)))
    row = slice(o.rowptr[c], o.rowptr[c + 1])
    o.rho[row][:14] = 0                                    # equal volumes: half of 28 bonds
    assert o.damage()[c] == pytest.approx(0.5, abs=1e-15)
    from paper_2309_11273_b200 import workloads
    wl = workloads.branching2d(nx=40, ny=20, steps=1)
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), precut=wl.precut)
    phi = o.damage().reshape(20, 40)
    assert np.all(phi[9:11, :17] > 0.35) and np.all(phi[9:11, :17] < 0.55)   # band next to the line
    assert np.all(phi[:, 26:] == 0.0) and np.all(phi[:6] == 0.0) and np.all(phi[14:] == 0.0)
    i, j = o.bond_pairs(intact=False)                      # symmetric pre-cut set
    assert set(zip(i.tolist(), j.tolist())) == set(zip(j.tolist(), i.tolist()))
    assert len(i) == 2 * len(wl.precut)


def test_fracture_run_monotone_symmetric_and_second_formulation():
    """Coarse config 2: phi never decreases, the mask stays symmetric every step, and the
    App. C pair-scatter formulation (oracle/pd_appc.py) gives the IDENTICAL break history."""
    from paper_2309_11273_b200 import workloads
    wl = workloads.branching2d(nx=32, ny=16, steps=1, sigma=60e6, ramp_steps=20)
    # App. C code has no body force; drive by initial velocity instead (same code paths for break)
    v0 = np.zeros((wl.n, 2)); v0[:, 1] = 40.0 * (wl.coords[:, 1] - wl.coords[:, 1].mean()) / 2e-3
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **{**wl.material_kwargs(), "ramp_time": 0.0},
                 precut=wl.precut, v0=v0)
    prev = o.damage().copy()
    for _ in range(40):
        o.step(5, log_breaks=True)
        phi = o.phi.copy()
        assert np.all(phi >= prev - 1e-15)
        prev = phi
        i, j = o.bond_pairs(intact=False)
        assert set(zip(i.tolist(), j.tolist())) == set(zip(j.tolist(), i.tolist()))
    assert len(o.break_log) > 50
    bonds, Xi, xi = pd_appc.bond_list(wl.coords, wl.horizon)
    cut = {(min(a, b), max(a, b)) for a, b in wl.precut.tolist()}
    co = np.array([0.0 if (a, b) in cut else 1.0 for a, b in bonds.tolist()])
    U, VEL, co2, breaks = pd_appc.run_explicit(wl.coords, wl.volumes, wl.horizon, o.A, o.K, o.G, wl.rho,
                                               wl.dt, 200, np.zeros((wl.n, 2)), v0,
                                               np.zeros((wl.n, 2), bool), s_c=wl.s_c, co_index=co)
    und = sorted({(s, min(i, j), max(i, j)) for s, i, j in o.break_log})
    assert und == sorted(breaks)
    assert np.max(np.abs(U - o.u)) <= 1e-11 * np.max(np.abs(o.u))


def test_second_formulation_config1_trajectory():
    """gather oracle vs App. C/B pair-scatter code after 2000 steps of config 1: <= 1e-12."""
    from paper_2309_11273_b200 import workloads
    wl = workloads.cantilever2d()
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, u0=wl.u0)
    o.step(2000)
    clamp = np.stack([(wl.flags & 1) != 0, (wl.flags & 2) != 0], axis=1)
    U, VEL, _, _ = pd_appc.run_explicit(wl.coords, wl.volumes, wl.horizon, o.A, o.K, o.G, wl.rho, wl.dt,
                                        2000, wl.u0, wl.v0, clamp)
    assert np.linalg.norm(U - o.u) <= 1e-12 * np.linalg.norm(o.u)
    assert np.linalg.norm(VEL - o.v) <= 1e-11 * np.linalg.norm(o.v)


# ---- scalars --------------------------------------------------------------------------------
def test_critical_stretch_and_literals():
    g = GOLD["s_c_spec_example"]
    assert scalars.critical_stretch(MODE_3D, 190e9, 0.25, 6.9e4, 1.5e-3) == pytest.approx(g["value"], rel=g["rtol"])
    from paper_2309_11273_b200 import workloads
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "scalars.json")))
    for name, row in gold.items():
        assert workloads.SCALARS[name]["dt"] == pytest.approx(row["dt"], rel=1e-12)
        assert workloads.SCALARS[name]["s_c"] == pytest.approx(row["s_c"], rel=1e-12)
        assert row["dt"] < 0.81 * row["dt_crit"] and row["dt_crit"] < row["delta_over_c"]  # reading C-8
    assert workloads.SCALARS["branching2d"]["s_c"] == pytest.approx(
        scalars.critical_stretch(MODE_PLANE_STRESS, 72e9, 0.22, 3.8, 3.015 * 2.5e-4), rel=1e-6)


# ---- variant: geometric extension (App. C) ------------------
def test_geometric_extension_pins():
    """e = ||xi + eta|| - ||xi||: (a) hand values on one bond (collinear stretch a -> e = a; transverse b -> e =
    sqrt(r^2 + b^2) - r while the linearized e is 0); (b) a FINITE rigid rotation leaves every bond length unchanged:
    e = 0, theta = 0, f = 0 to roundoff, where the linearized model gives a spurious force; (c) e_geo - e_lin is of
    second order in eta; (d) the App. C pair-scatter code with the extension as printed gives the same force."""
    r, a, b = 0.5, 1e-3, 2e-3
    x2 = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
    for u1, e_geo, e_lin in (([a, 0, 0], a, a), ([0, b, 0], np.sqrt(r * r + b * b) - r, 0.0)):
        u = np.array([[0, 0, 0], u1], float)
        og = make(x2, 3, MODE_3D, 1.0, extension="geometric", u0=u)
        ol = make(x2, 3, MODE_3D, 1.0, u0=u)
        assert og.extension()[0] == pytest.approx(e_geo, rel=1e-12, abs=1e-18)
        assert ol.extension()[0] == pytest.approx(e_lin, rel=1e-12, abs=1e-18)
    # (b) finite rotation by 30 degrees about z plus a translation
    x = lattice((7, 6, 5))
    c, s_ = np.cos(np.pi / 6), np.sin(np.pi / 6)
    Rm = np.array([[c, -s_, 0], [s_, c, 0], [0, 0, 1.0]])
    u = x @ Rm.T - x + np.array([0.3, -0.2, 0.1])
    og = make(x, 3, MODE_3D, 3.015, extension="geometric", u0=u)
    ol = make(x, 3, MODE_3D, 3.015, u0=u)
    fg, fl = og.force_density(), ol.force_density().copy()
    scale = np.max(np.abs(fl))
    assert np.max(np.abs(og.e)) <= 1e-13 * 3.0 and np.max(np.abs(og.theta)) <= 1e-12
    assert np.max(np.abs(fg)) <= 1e-10 * scale and scale > 0
    # (c) second-order agreement: halving eta quarters the difference
    rng = np.random.default_rng(3)
    w = rng.standard_normal(x.shape)
    d = []
    for amp in (1e-3, 5e-4):
        eg = make(x, 3, MODE_3D, 3.015, extension="geometric", u0=amp * w).extension().copy()
        el = make(x, 3, MODE_3D, 3.015, u0=amp * w).extension().copy()
        d.append(np.max(np.abs(eg - el)))
    assert d[0] / d[1] == pytest.approx(4.0, rel=0.02) and d[0] < 1e-4
    # (d) second formulation: App. C exactly as printed
    x = lattice((6, 5)) * 1e-3
    u = 1e-5 * rng.standard_normal(x.shape)
    vol = np.full(len(x), 1e-9)
    og = make(x, 2, MODE_PLANE_STRESS, 3.015e-3, vol=vol, extension="geometric", u0=u)
    f = og.force_density()
    bonds, Xi, xi = pd_appc.bond_list(x, 3.015e-3)
    m = pd_appc.weighted_volume(len(x), bonds, xi, vol)
    PDF, _ = pd_appc.pd_force(u, vol, bonds, m, xi, Xi, np.ones(len(bonds)), og.A, og.K, og.G, geometric=True)
    assert np.max(np.abs(PDF / vol[:, None] - f)) <= 1e-12 * np.max(np.abs(f))


def test_geometric_break_and_run():
    """the failure stretch of the variant is s = e_geo / xbar; a transverse displacement that stretches the bond past
    s_c breaks it although the linearized stretch is 0; the stepper conserves momentum like the linearized one"""
    r, s_c = 1.0, 1e-3
    b = r * np.sqrt((1 + s_c) ** 2 - 1) * (1 + 1e-9)          # ||xi + eta|| = r (1 + s_c) (1 + ...)
    x = np.array([[0.0, 0.0], [r, 0.0]])
    u = np.array([[0.0, 0.0], [0.0, b]])
    og = make(x, 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, extension="geometric", u0=u)
    ol = make(x, 2, MODE_PLANE_STRAIN, 1.5, s_c=s_c, u0=u)
    assert og.break_bonds()[0] == 2 and ol.break_bonds()[0] == 0
    x = lattice((9, 7)) * 1e-3
    rng = np.random.default_rng(5)
    o = make(x, 2, MODE_PLANE_STRESS, 3.015e-3, vol=np.full(len(x), 1e-9), extension="geometric", dt=5e-8,
             v0=rng.standard_normal(x.shape))
    p0 = o.v.sum(0).copy()
    o.step(50)
    assert np.allclose(o.v.sum(0), p0, rtol=0, atol=1e-12 * np.abs(o.v).sum())


# ---- NEXT row f1: adaptive dynamic relaxation --------------------------
def test_adr_converges_to_direct_solve():
    """ADR on the oracle's force: (a) 1-dof spring analogue (two nodes, one clamped) -> U = F/k; (b) zero load -> 0;
    (c) a small 3-D bar, one end clamped, body force on the other end layer AND a prescribed-displacement variant:
    the converged U equals the direct dense solve of K U = F (K assembled from the linear oracle force) to 1e-6."""
    from oracle.pd_adr import ADROracle, dense_stiffness
    # (a) two nodes on the x axis, node 0 clamped, body force b on node 1 (x only; y clamped on both)
    x = np.array([[0.0, 0.0], [1.0, 0.0]])
    fl = np.array([3, 2 | 64], np.uint8)
    val = np.array([[0.0, 0.0], [2.5, 0.0]])
    o = make(x, 2, MODE_PLANE_STRAIN, 1.5, E=3.0, nu=0.25, flags=fl, value=val)
    K = dense_stiffness(o)
    k = K[2, 2]
    adr = ADROracle(o, lam=0.3 * k)
    adr.iterate(400)
    assert o.u[1, 0] == pytest.approx(2.5 / k, rel=1e-8) and np.all(o.u[0] == 0)
    # (b) zero load
    o = make(x, 2, MODE_PLANE_STRAIN, 1.5, E=3.0, nu=0.25, flags=np.array([3, 2], np.uint8))
    ADROracle(o, lam=1.0).iterate(5)
    assert np.all(o.u == 0.0)
    # (c) bar 10 x 4 x 4, clamp x < 2 cells
    xb = lattice((10, 4, 4))
    ix = xb[:, 0]
    fl = np.zeros(len(xb), np.uint8)
    fl[ix < 2] = 7
    val = np.zeros_like(xb)
    for mode in ("force", "displacement"):
        f2, v2 = fl.copy(), val.copy()
        if mode == "force":
            f2[ix > 8.5] |= 64
            v2[ix > 8.5] = [1e-3, 2e-4, 0.0]
        o = make(xb, 3, MODE_3D, 2.015, E=1.0, nu=0.25, flags=f2, value=v2)
        K = dense_stiffness(o)
        assert np.max(np.abs(K - K.T)) <= 1e-12 * np.max(np.abs(K))
        lam = 1.05 * 0.25 * np.linalg.eigvalsh(K)[-1]
        fixed = np.repeat(f2 & 7, 3).reshape(-1, 3)
        fixed = np.stack([(f2 & (1 << k_)) != 0 for k_ in range(3)], axis=1).reshape(-1)
        rhs = np.where(((f2 & 64) != 0)[:, None], v2, 0.0).reshape(-1)
        uc = np.zeros(len(rhs))
        if mode == "displacement":        # drive the end layer to u_x = 1e-3 in 50 increments, then relax
            f2[ix > 8.5] |= 8
            v2[ix > 8.5] = [2e-5, 0.0, 0.0]
            o = make(xb, 3, MODE_3D, 2.015, E=1.0, nu=0.25, flags=f2, value=v2)
            adr = ADROracle(o, lam)
            adr.iterate(50)
            o.value[:] = 0.0              # hold
            adr.iterate(3000)
            drv = np.stack([(f2 & (8 << k_)) != 0 for k_ in range(3)], axis=1).reshape(-1)
            uc[drv] = 50 * 2e-5
            fixed = fixed | drv
        else:
            adr = ADROracle(o, lam)
            adr.iterate(3000)
        free = ~fixed
        usol = uc.copy()
        usol[free] = np.linalg.solve(K[np.ix_(free, free)], rhs[free] - K[np.ix_(free, fixed)] @ uc[fixed])
        err = np.linalg.norm(o.u.reshape(-1) - usol) / np.linalg.norm(usol)
        assert err <= 1e-6, (mode, err)
        assert max(adr.c_hist) > 0.0      # the adaptive damping was active
