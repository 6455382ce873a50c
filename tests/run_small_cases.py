"""Runs the small parity cases once on the default code path (no oracle): the workload of the compute-sanitizer
passes recorded in profiles/r02_sanitizer.md:

    compute-sanitizer --tool memcheck  python tests/run_small_cases.py
    compute-sanitizer --tool racecheck python tests/run_small_cases.py

(not collected by pytest; prints one line per case with a checksum so that a run can be compared with a plain one)"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    from paper_2309_11273_b200 import pd, workloads as W
    cases = {
        "config1": (W.cantilever2d(), 40),
        "config2_small": (W.branching2d(nx=100, ny=44, steps=600), 260),     # bonds break from step ~200 on
        "config3_small": (W.impact2d(nx=72, ny=72), 120),
        "config4_small": (W.block3d(nx=37, ny=13, nz=11), 12),               # jittered: per-bond-geometry lattice kernels
        "config5_small": (W.cylinder3d(r_cells=9, l_cells=34, omega=400.0), 40),   # uniform-lattice kernels, TMA planes, breaking
    }
    for name, (wl, nsteps) in cases.items():
        sim = pd.Sim.from_workload(wl)
        sim.step(nsteps)
        st = sim.get_stats()
        u, phi = sim.get_u(), sim.get_damage()
        print(f"{name}: layout {sim.get_layout()['layout']} steps {st['step']} broken {st['n_broken_directed']} "
              f"sum|u| {np.abs(u).sum():.12e} max phi {phi.max():.6f}", flush=True)
        sim.destroy()


if __name__ == "__main__":
    main()
