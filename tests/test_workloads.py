"""Host-side checks of the synthetic input generators (geometry only) against SURVEY.md 8's
exact lattice counts and against the oracle's family definition."""
import numpy as np
import pytest

from oracle.pd_oracle import PDOracle, family
from paper_2309_11273_b200 import workloads as W


def test_cylinder_slice_count():
    wl = W.cylinder3d(r_cells=50, l_cells=2, steps=1)
    assert wl.meta["slice_nodes"] == 7860 and wl.n == 2 * 7860      # 7 860/slice


def test_config_shapes_small():
    for wl, z in [(W.cantilever2d(), 24076)]:
        rp, _ = family(wl.coords, wl.horizon)
        assert rp[-1] == z
    wl = W.block3d(nx=12, ny=8, nz=8)
    rp, _ = family(wl.coords, wl.horizon)                            # jitter keeps the lattice topology
    rq, _ = family(np.round(wl.coords / wl.dx - 0.5) + 0.5, 3.015)
    assert np.array_equal(rp, rq)
    assert np.max(np.abs(wl.coords / wl.dx - 0.5 - np.round(wl.coords / wl.dx - 0.5))) <= 1e-3 + 1e-12


@pytest.mark.parametrize("make", [lambda: W.branching2d(nx=40, ny=16), lambda: W.impact2d(nx=32, ny=32),
                                  lambda: W.cylinder3d(r_cells=8, l_cells=24)])
def test_precut_pairs_are_bonds_and_cross(make):
    wl = make()
    assert len(wl.precut) > 0
    assert len({(min(a, b), max(a, b)) for a, b in wl.precut.tolist()}) == len(wl.precut)  # each once
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), precut=wl.precut)  # raises if not a bond
    assert (o.rho == 0).sum() == 2 * len(wl.precut)
    xa, xb = wl.coords[wl.precut[:, 0]], wl.coords[wl.precut[:, 1]]
    if wl.dim == 2:
        lines = ([wl.meta["ny"] // 2] if wl.name == "branching2d" else [wl.meta["r1"], wl.meta["r2"]])
        yl = np.array(lines) * wl.dx
        crossed = np.any([(np.minimum(xa[:, 1], xb[:, 1]) < y) & (np.maximum(xa[:, 1], xb[:, 1]) > y) for y in yl], axis=0)
        assert crossed.all()
        # brute force the same rule in floating point on every bond
        i, j = o.bond_pairs()
        keep = i < j
        i, j = i[keep], j[keep]
        tipx = (wl.meta["nx"] // (2 if wl.name == "branching2d" else 4)) * wl.dx
        cnt = 0
        for y in yl:
            ya, yb = wl.coords[i, 1], wl.coords[j, 1]
            cr = (np.minimum(ya, yb) < y) & (np.maximum(ya, yb) > y)
            t = (y - ya[cr]) / (yb[cr] - ya[cr])
            xc = wl.coords[i[cr], 0] + t * (wl.coords[j[cr], 0] - wl.coords[i[cr], 0])
            cnt += int((xc <= tipx + 1e-12).sum())
        assert cnt == len(wl.precut)
    else:
        L = wl.meta["l_cells"] * wl.dx
        g = lambda x: x[:, 2] - x[:, 1] - (0.5 * L + 0.5 * wl.dx)
        assert np.all(g(xa) * g(xb) < 0)
        i, j = o.bond_pairs()
        keep = i < j
        i, j = i[keep], j[keep]
        ga, gb = g(wl.coords[i]), g(wl.coords[j])
        cr = ga * gb < 0
        t = ga[cr] / (ga[cr] - gb[cr])
        xc = wl.coords[i[cr], 0] + t * (wl.coords[j[cr], 0] - wl.coords[i[cr], 0])
        depth = round(0.4 * wl.meta["r_cells"]) * wl.dx
        assert int((xc >= wl.meta["r_cells"] * wl.dx - depth - 1e-12).sum()) == len(wl.precut)


def test_boundary_sets():
    wl = W.cylinder3d(r_cells=6, l_cells=20)
    z = wl.coords[:, 2] / wl.dx
    assert np.all((wl.flags[z < 3] & 7) == 7) and np.all((wl.flags[z > 17] & 56) == 56)
    assert np.all((wl.flags[(z > 3) & (z < 17)]) == 0)
    top = z > 17
    assert np.allclose(wl.value[top, 0], -100.0 * wl.coords[top, 1]) and np.allclose(wl.value[top, 2], 0)
    wl = W.impact2d(nx=32, ny=32)
    drv = (wl.flags & 8) != 0
    assert drv.sum() == 3 * (wl.meta["r2"] - wl.meta["r1"]) and np.all(wl.value[drv, 0] == 16.5)
    wl = W.cantilever2d()
    assert sorted(wl.meta["perm"].tolist()) == list(range(1000)) and not np.array_equal(wl.meta["perm"], np.arange(1000))
