"""Seeded synthetic input generators for the five workloads of BASELINE.json (+5').

This module serves BOTH the CUDA library and the CPU oracle and therefore holds none of the
method's arithmetic: it only lays out nodes, volumes, boundary flags/values, pre-cut pair lists
and initial fields, and carries the scalar inputs s_c and dt as LITERALS (written by
oracle/derive_scalars.py).  It imports neither the binding nor
the oracle.

Stand-ins, not the paper's models: the paper uses no public dataset; its
examples are node-on-boundary grids of other sizes/materials.  These inputs have the shapes,
family sizes (28 in 2D, 122 in 3D at delta = 3.015 dx), boundary conditions and pre-crack
structure of Ex. 1-4, per SURVEY.md 8(d) and readings C-13..C-21.

Every generator accepts reduced grid sizes (same dx, same material, same dt and s_c) so the
parity tests can run the same recipe at sizes the oracle finishes in seconds.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

MODE_3D, MODE_PLANE_STRESS, MODE_PLANE_STRAIN = 0, 1, 2
CLAMP_X, CLAMP_Y, CLAMP_Z = 1, 2, 4
PRESC_X, PRESC_Y, PRESC_Z = 8, 16, 32
BODY_FORCE, NO_FAIL = 64, 128

M_RATIO = 3.015  # horizon / dx in every config (BASELINE.json)

# ---- scalar inputs, literals written by `python -m oracle.derive_scalars` ----------------
# dt  = 0.8 * 2/omega_max of the intact discrete operator (reading C-8; Eq. 2.13's delta/c'
#       is not a sufficient bound), per config family (depends on material, mode, dx only).
# s_c = Eq. 1.26 / 1.28 with beta, beta' AS PRINTED in Eqs. 1.27 / 1.29 (reading C-9).
SCALARS = {
    "cantilever2d": {"dt": 2.6825e-07, "s_c": 0.0},
    "branching2d": {"dt": 6.7387e-08, "s_c": 2.764611e-04},
    "impact2d": {"dt": 1.4825e-07, "s_c": 8.890326e-03},
    "block3d": {"dt": 2.4641e-07, "s_c": 0.0},
    "cylinder3d": {"dt": 6.1604e-08, "s_c": 6.451128e-04},
}

GLASS = dict(E=72e9, nu=0.22, rho=2440.0)
STEEL = dict(E=190e9, nu=0.3, rho=8000.0)


@dataclass
class Workload:
    name: str
    dim: int
    mode: int
    coords: np.ndarray          # (N, dim) float64
    volumes: np.ndarray         # (N,) float64
    horizon: float
    E: float
    nu: float
    rho: float
    s_c: float                  # 0 => fracture off
    dt: float
    ramp_time: float
    flags: np.ndarray           # (N,) uint8
    value: np.ndarray           # (N, dim) float64: prescribed velocity or body-force density
    precut: np.ndarray          # (P, 2) int32 user-index pairs (each undirected bond once)
    u0: np.ndarray              # (N, dim)
    v0: np.ndarray              # (N, dim)
    steps: int
    dx: float
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.coords.shape[0])

    def material_kwargs(self) -> dict:
        return dict(dim=self.dim, mode=self.mode, E=self.E, nu=self.nu, rho=self.rho,
                    dt=self.dt, s_c=self.s_c, ramp_time=self.ramp_time)


# ---- lattice helpers (geometry only) ------------------------------------------------------
def _lattice_offsets(dim: int) -> np.ndarray:
    """Integer lattice offsets o != 0 with |o|^2 <= 9 (< 3.015^2 = 9.09 < 10): the neighbours a
    lattice node has at horizon 3.015 dx.  Used only to enumerate candidate pre-cut pairs."""
    r = np.arange(-3, 4)
    g = np.stack(np.meshgrid(*([r] * dim), indexing="ij"), axis=-1).reshape(-1, dim)
    n2 = np.sum(g * g, axis=1)
    return g[(n2 > 0) & (n2 <= 9)]


def _grid2d(nx, ny, dx):
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")  # node id = iy*nx + ix
    ix, iy = ix.reshape(-1), iy.reshape(-1)
    coords = np.stack([(ix + 0.5) * dx, (iy + 0.5) * dx], axis=1)
    return ix, iy, coords


def _precut_horizontal(nx, ny, row_line, tip_half_x):
    """Pairs (a<b) of 2D lattice bonds crossing the line y = row_line*dx (a cell face) at a
    point x_c <= tip (tip inclusive).  Exact integer arithmetic in half-cell units
    (reading C-16): X = 2 ix + 1, Y = 2 iy + 1, line Y_l = 2 row_line, tip X_t = tip_half_x."""
    pairs = []
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    ix, iy = ix.reshape(-1), iy.reshape(-1)
    Yl = 2 * row_line
    for ox, oy in _lattice_offsets(2):
        if oy <= 0:
            continue                      # take each undirected bond once, from below to above
        jx, jy = ix + ox, iy + oy
        ok = (jx >= 0) & (jx < nx) & (jy < ny) & (iy < row_line) & (jy >= row_line)
        Xa, Ya = 2 * ix[ok] + 1, 2 * iy[ok] + 1
        DX, DY = 2 * ox, 2 * oy
        # x_c = Xa + (Yl - Ya) * DX / DY  <= X_t   <=>   Xa*DY + (Yl-Ya)*DX <= X_t*DY  (DY > 0)
        hit = Xa * DY + (Yl - Ya) * DX <= tip_half_x * DY
        a = (iy[ok] * nx + ix[ok])[hit]
        b = (jy[ok] * nx + jx[ok])[hit]
        pairs.append(np.stack([a, b], axis=1))
    return np.concatenate(pairs).astype(np.int32) if pairs else np.zeros((0, 2), np.int32)


# ---- config 1 ------------------------------------------------------------------------------
def cantilever2d(nx=100, ny=10, steps=2000, seed=1234, shuffle=True) -> Workload:
    """Config 1: 2D plane-stress cantilever, no fracture, shuffled node order (C-13, C-20)."""
    dx, t = 1e-3, 1e-3
    ix, iy, coords = _grid2d(nx, ny, dx)
    n = nx * ny
    L = nx * dx
    u0 = np.zeros((n, 2))
    u0[:, 1] = 1e-5 * (coords[:, 0] / L) ** 2
    flags = np.zeros(n, np.uint8)
    flags[ix < 3] = CLAMP_X | CLAMP_Y
    u0[ix < 3] = 0.0
    perm = np.random.default_rng(seed).permutation(n) if shuffle else np.arange(n)
    sc = SCALARS["cantilever2d"]
    return Workload("cantilever2d", 2, MODE_PLANE_STRESS, coords[perm].copy(), np.full(n, dx * dx * t),
                    M_RATIO * dx, **GLASS, s_c=0.0, dt=sc["dt"], ramp_time=0.0, flags=flags[perm].copy(),
                    value=np.zeros((n, 2)), precut=np.zeros((0, 2), np.int32), u0=u0[perm].copy(),
                    v0=np.zeros((n, 2)), steps=steps, dx=dx, meta=dict(nx=nx, ny=ny, perm=perm))


# ---- config 2 ------------------------------------------------------------------------------
def branching2d(nx=400, ny=160, steps=2000, sigma=12e6, ramp_steps=500) -> Workload:
    """Config 2: pre-cracked plate under ramped traction (C-14, C-15, C-16, C-21)."""
    dx, t = 2.5e-4, 1e-3
    ix, iy, coords = _grid2d(nx, ny, dx)
    n = nx * ny
    flags = np.zeros(n, np.uint8)
    value = np.zeros((n, 2))
    top, bot = iy == ny - 1, iy == 0
    flags[top | bot] = BODY_FORCE
    value[top, 1] = +sigma / dx          # force density N/m^3 on the outermost node row
    value[bot, 1] = -sigma / dx
    precut = _precut_horizontal(nx, ny, ny // 2, 2 * (nx // 2))
    sc = SCALARS["branching2d"]
    return Workload("branching2d", 2, MODE_PLANE_STRESS, coords, np.full(n, dx * dx * t), M_RATIO * dx,
                    **GLASS, s_c=sc["s_c"], dt=sc["dt"], ramp_time=ramp_steps * sc["dt"], flags=flags,
                    value=value, precut=precut, u0=np.zeros((n, 2)), v0=np.zeros((n, 2)), steps=steps,
                    dx=dx, meta=dict(nx=nx, ny=ny))


# ---- config 3 ------------------------------------------------------------------------------
def impact2d(nx=400, ny=400, steps=3000, vbar=16.5) -> Workload:
    """Config 3: edge-impact plate with two parallel pre-notches (C-15, C-16, C-17)."""
    dx, t = 5e-4, 1.0
    ix, iy, coords = _grid2d(nx, ny, dx)
    n = nx * ny
    r1, r2 = (3 * ny) // 8, (5 * ny) // 8          # notch lines y = r*dx (0.075 / 0.125 m at 400)
    tip = 2 * (nx // 4)                            # notch length nx/4 cells (0.05 m at 400)
    precut = np.concatenate([_precut_horizontal(nx, ny, r1, tip), _precut_horizontal(nx, ny, r2, tip)])
    flags = np.zeros(n, np.uint8)
    value = np.zeros((n, 2))
    drv = (ix < 3) & (iy >= r1) & (iy < r2)
    flags[drv] = PRESC_X
    value[drv, 0] = vbar
    v0 = np.zeros((n, 2))
    v0[drv, 0] = vbar
    sc = SCALARS["impact2d"]
    return Workload("impact2d", 2, MODE_PLANE_STRAIN, coords, np.full(n, dx * dx * t), M_RATIO * dx,
                    **STEEL, s_c=sc["s_c"], dt=sc["dt"], ramp_time=0.0, flags=flags, value=value,
                    precut=precut, u0=np.zeros((n, 2)), v0=v0, steps=steps, dx=dx,
                    meta=dict(nx=nx, ny=ny, r1=r1, r2=r2))


# ---- config 4 ------------------------------------------------------------------------------
def block3d(nx=200, ny=40, nz=40, steps=1000, seed=4321, amp=1e-5, jitter=1e-3) -> Workload:
    """Config 4: 3D cantilever block, jittered lattice (jitter = 0: plain lattice), bending + torsion start (C-18)."""
    dx = 1e-3
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ix, iy, iz = ix.reshape(-1), iy.reshape(-1), iz.reshape(-1)   # id = (iz*ny + iy)*nx + ix
    n = nx * ny * nz
    coords = np.stack([(ix + 0.5) * dx, (iy + 0.5) * dx, (iz + 0.5) * dx], axis=1)
    if jitter != 0.0:
        coords = coords + np.random.default_rng(seed).uniform(-jitter * dx, jitter * dx, size=(n, 3))
    L, yc, zc, Rh = nx * dx, 0.5 * ny * dx, 0.5 * nz * dx, 0.5 * ny * dx
    x, y, z = coords[:, 0], coords[:, 1], coords[:, 2]
    u0 = np.zeros((n, 3))
    u0[:, 1] = amp * (x / L) ** 2 - amp * (x / L) * (z - zc) / Rh
    u0[:, 2] = amp * (x / L) * (y - yc) / Rh
    flags = np.zeros(n, np.uint8)
    flags[ix < 3] = CLAMP_X | CLAMP_Y | CLAMP_Z
    u0[ix < 3] = 0.0
    sc = SCALARS["block3d"]
    return Workload("block3d", 3, MODE_3D, coords, np.full(n, dx ** 3), M_RATIO * dx, **GLASS, s_c=0.0,
                    dt=sc["dt"], ramp_time=0.0, flags=flags, value=np.zeros((n, 3)),
                    precut=np.zeros((0, 2), np.int32), u0=u0, v0=np.zeros((n, 3)), steps=steps, dx=dx,
                    meta=dict(nx=nx, ny=ny, nz=nz, jitter=jitter))


# ---- config 5 / 5' -------------------------------------------------------------------------
def cylinder3d(r_cells=50, l_cells=400, steps=2000, omega=100.0, notch_depth_cells=None) -> Workload:
    """Config 5: notched cylinder under torsion (C-19).  r_cells = R/dx, l_cells = L/dx (even).
    Full size: r_cells=50, l_cells=400 (3 144 000 nodes); 5': l_cells=160 (1 257 600 nodes)."""
    assert l_cells % 2 == 0
    dx = 2.5e-4
    Rc, Lc = r_cells, l_cells
    depth = int(round(0.4 * Rc)) if notch_depth_cells is None else notch_depth_cells  # 5 mm of 12.5
    # slice: lattice points with x^2 + y^2 <= R^2, centred, exact in half-cell integers
    g = np.arange(2 * Rc)
    hx, hy = np.meshgrid(2 * g + 1 - 2 * Rc, 2 * g + 1 - 2 * Rc, indexing="xy")
    inside = hx * hx + hy * hy <= (2 * Rc) ** 2
    sid = -np.ones(inside.shape, np.int64)
    sid[inside] = np.arange(int(inside.sum()))          # slice-local id, raster (y, x)
    sx, sy = hx[inside], hy[inside]                     # half-cell centred coords per slice node
    ns = sx.size
    n = ns * Lc
    iz = np.repeat(np.arange(Lc), ns)
    X = np.tile(sx, Lc)
    Y = np.tile(sy, Lc)
    coords = np.stack([X * (0.5 * dx), Y * (0.5 * dx), (iz + 0.5) * dx], axis=1)
    flags = np.zeros(n, np.uint8)
    value = np.zeros((n, 3))
    bot, top = iz < 3, iz >= Lc - 3
    flags[bot] = CLAMP_X | CLAMP_Y | CLAMP_Z | NO_FAIL
    flags[top] = PRESC_X | PRESC_Y | PRESC_Z | NO_FAIL
    value[top, 0] = -omega * coords[top, 1]
    value[top, 1] = +omega * coords[top, 0]
    v0 = np.zeros((n, 3))
    v0[top] = value[top]
    # notch: bonds crossing the plane z - y = L/2 + dx/2 at a point with x >= R - depth.
    # half-cell integers: gval = 2 iz + 1 - Yh - (Lc + 1), odd for even Lc => never 0.
    ixg = (sx + 2 * Rc - 1) // 2
    iyg = (sy + 2 * Rc - 1) // 2
    Xd = 2 * (Rc - depth)
    pairs = []
    for ox, oy, oz in _lattice_offsets(3):
        if (oz, oy, ox) <= (0, 0, 0):
            continue                                   # each undirected bond once
        jx, jy = ixg + ox, iyg + oy
        okxy = (jx >= 0) & (jx < 2 * Rc) & (jy >= 0) & (jy < 2 * Rc)
        jsid = np.where(okxy, sid[np.clip(jy, 0, 2 * Rc - 1), np.clip(jx, 0, 2 * Rc - 1)], -1)
        sel = np.nonzero(jsid >= 0)[0]
        if sel.size == 0:
            continue
        # plane crossing depends on iz only through 2*iz; restrict to the slab of iz that can cross
        for za in range(max(0, Lc // 2 - Rc - 4), min(Lc, Lc // 2 + Rc + 5)):
            zb = za + oz
            if zb < 0 or zb >= Lc:
                continue
            ga = 2 * za + 1 - sy[sel] - (Lc + 1)
            gb = 2 * zb + 1 - (sy[sel] + 2 * oy) - (Lc + 1)
            cross = (ga < 0) != (gb < 0)
            if not cross.any():
                continue
            Xa, Xb = sx[sel], sx[sel] + 2 * ox
            den = ga - gb
            num = Xa * den + ga * (Xb - Xa)            # x_c * den
            deep = np.where(den > 0, num >= Xd * den, num <= Xd * den)
            hit = cross & deep
            if hit.any():
                a = za * ns + np.arange(ns)[sel][hit]
                b = zb * ns + jsid[sel][hit]
                pairs.append(np.stack([a, b], axis=1))
    precut = (np.concatenate(pairs).astype(np.int32) if pairs else np.zeros((0, 2), np.int32))
    sc = SCALARS["cylinder3d"]
    return Workload("cylinder3d", 3, MODE_3D, coords, np.full(n, dx ** 3), M_RATIO * dx, **GLASS,
                    s_c=sc["s_c"], dt=sc["dt"], ramp_time=0.0, flags=flags, value=value, precut=precut,
                    u0=np.zeros((n, 3)), v0=v0, steps=steps, dx=dx,
                    meta=dict(r_cells=Rc, l_cells=Lc, slice_nodes=int(ns), omega=omega))


CONFIGS = {
    "config1": cantilever2d,
    "config2": branching2d,
    "config3": impact2d,
    "config4": block3d,
    "config5": cylinder3d,
    "config5p": lambda **kw: cylinder3d(l_cells=160, **kw),
}
