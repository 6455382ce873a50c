"""Writes the scalar literals carried by paper_2309_11273_b200/workloads.py (SCALARS) and
tests/golden/scalars.json.  Calls only oracle/ (+ the geometry generators).

  python -m oracle.derive_scalars            # prints the table, rewrites tests/golden/scalars.json

dt: reading C-8.  Eq. 2.13's delta/c' is not a sufficient bound
for this discretisation, so "critical" is 2/omega_max of the intact discrete operator
u -> -f(u)/rho (f from oracle steps 6-8), found by power iteration from a seeded start on a
reduced-size instance of each config (same dx, material, mode; omega_max is a local lattice
property).  dt = 0.8 * 2/omega_max, rounded DOWN to 5 significant digits.
s_c: Eq. 1.26 / 1.28 with the constants of Eqs. 1.27 / 1.29 as printed (reading C-9).
"""
from __future__ import annotations

import json
import math
import os
import sys

import numpy as np

from oracle import scalars
from oracle.pd_oracle import PDOracle
from paper_2309_11273_b200 import workloads as W


def omega_max(wl, iters=400, seed=7):
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs())  # no BC, intact
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((wl.n, wl.dim))
    lam = 0.0
    for _ in range(iters):
        x /= np.linalg.norm(x)
        y = -o.force_density(x) / wl.rho
        lam = float(np.sum(x * y))          # Rayleigh quotient (operator symmetric for uniform V)
        x = y.copy()
    return math.sqrt(lam)


def round_down(x, sig=5):
    e = math.floor(math.log10(x)) - (sig - 1)
    return float(f"{math.floor(x / 10 ** e) * 10 ** e:.{sig - 1}e}")


def main():
    reduced = {
        "cantilever2d": W.cantilever2d(),                      # full size (1000 nodes)
        "branching2d": W.branching2d(nx=120, ny=60),
        "impact2d": W.impact2d(nx=96, ny=96),
        "block3d": W.block3d(nx=30, ny=16, nz=16),
        "cylinder3d": W.cylinder3d(r_cells=12, l_cells=40),
    }
    G0 = {"branching2d": 3.8, "impact2d": 2.2e4, "cylinder3d": 8.0}
    out = {}
    for name, wl in reduced.items():
        wm = omega_max(wl)
        crit = 2.0 / wm
        bound = scalars.wave_speed_bound(wl.E, wl.nu, wl.rho, wl.horizon)
        row = {"dt_crit": crit, "dt": round_down(0.8 * crit), "delta_over_c": bound,
               "ratio_crit_over_bound": crit / bound, "s_c": 0.0}
        if name in G0:
            row["s_c"] = float(f"{scalars.critical_stretch(wl.mode, wl.E, wl.nu, G0[name], wl.horizon):.7g}")
            row["s_c_integrated_beta"] = scalars.critical_stretch(wl.mode, wl.E, wl.nu, G0[name], wl.horizon,
                                                                  "integrated")
        out[name] = row
    # the reduced cylinder is small enough for its surface to soften omega_max; the full-size
    # cylinder interior is the block's lattice, so take the smaller (safer) crit/bound ratio
    r3 = min(out["block3d"]["ratio_crit_over_bound"], out["cylinder3d"]["ratio_crit_over_bound"])
    out["cylinder3d"]["ratio_used"] = r3
    out["cylinder3d"]["dt"] = round_down(0.8 * r3 * out["cylinder3d"]["delta_over_c"])
    for name, row in out.items():
        print(name, json.dumps(row))
    path = os.path.join(os.path.dirname(__file__), "..", "tests", "golden", "scalars.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1, sort_keys=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
