"""Full-size, stated-step parity of one workload against the oracle (not collected by pytest: the oracle needs about
20 minutes of 16 host cores for the 6.3e9 node-steps of config 5).  The record of the runs is profiles/r02_parity_full.md.

    python tests/run_full_parity.py --workload config5 [--checkpoints 4] [--out gpurun_out/parity_full_config5.json]

Runs the workload of BASELINE.json at its stated size for its stated number of steps on the CUDA path (through the C
ABI, default layout and launch configuration: what bench.py times) and on the oracle, and compares at every checkpoint
  * the set of broken directed bonds (user index pairs; must be identical),
  * u and v (relative L2) and the damage field (max abs difference),
and reports the oracle's count of bonds that broke within 1e-9 relative of s_c (near-threshold events: a difference in
the broken sets would have to be explained by one of them).  Exit code 0 only if every checkpoint matches.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

TOL_FIELD = 1e-9        # relative L2 of u, v on fracture runs
TOL_FIELD_NO_FRACTURE = 1e-10   # north star, configs without fracture
TOL_DAMAGE = 1e-12


def _rel(a, b):
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def _broken_keys(n, rowptr, col, broken):
    """sorted int64 keys i * n + j of the broken directed bonds"""
    idx = np.flatnonzero(broken)
    i = np.searchsorted(rowptr, idx, side="right") - 1
    keys = i.astype(np.int64) * n + col[idx].astype(np.int64)
    keys.sort()
    return keys


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config5")
    ap.add_argument("--checkpoints", type=int, default=4)
    ap.add_argument("--steps", type=int, default=None, help="default: the workload's stated step count")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    from oracle.pd_oracle import PDOracle, num_threads
    from paper_2309_11273_b200 import pd, workloads as W
    wl = W.CONFIGS[args.workload]()
    steps = args.steps or wl.steps
    t0 = time.perf_counter()
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                 precut=wl.precut, u0=wl.u0, v0=wl.v0)
    t_obuild = time.perf_counter() - t0
    sim = pd.Sim.from_workload(wl)
    lay = sim.get_layout()
    rec = {"workload": f"{args.workload}:{wl.name}", "nodes": wl.n, "directed_bonds": o.Z, "steps": steps,
           "layout": lay["layout"], "oracle_threads": num_threads(), "oracle_build_seconds": t_obuild, "checkpoints": []}
    assert lay["n_directed_bonds"] == o.Z, "the two families differ"
    print(f"{rec['workload']}: n={wl.n} Z={o.Z} layout={lay['layout']} steps={steps} "
          f"(oracle build {t_obuild:.1f} s, {rec['oracle_threads']} threads)", flush=True)
    tol = TOL_FIELD if wl.s_c > 0 else TOL_FIELD_NO_FRACTURE
    rec["tolerance_rel_l2"] = tol
    ok, done, t_gpu, t_cpu = True, 0, 0.0, 0.0
    marks = [steps * (c + 1) // args.checkpoints for c in range(args.checkpoints)]
    for mark in marks:
        chunk = mark - done
        t0 = time.perf_counter()
        sim.step(chunk)
        st = sim.get_stats()            # synchronises
        t_gpu += time.perf_counter() - t0
        t0 = time.perf_counter()
        o.step(chunk)
        t_cpu += time.perf_counter() - t0
        done = mark
        rp, col, intact = sim.get_bond_mask()
        kg = _broken_keys(wl.n, rp, col, intact == 0)
        ko = _broken_keys(wl.n, o.rowptr, o.col, o.rho == 0)
        del rp, col, intact
        same = kg.size == ko.size and bool(np.array_equal(kg, ko))
        symdiff = 0 if same else int(np.setxor1d(kg, ko, assume_unique=True).size)
        eu, ev = _rel(sim.get_u(), o.u), _rel(sim.get_v(), o.v)
        dphi = float(np.abs(sim.get_damage() - o.damage()).max())
        cp = {"step": done, "broken_directed_cuda": int(kg.size), "broken_directed_oracle": int(ko.size),
              "symmetric_difference": symdiff, "near_threshold_events": int(o.near_total), "rel_l2_u": eu, "rel_l2_v": ev,
              "max_abs_damage_diff": dphi, "stats_broken": st["n_broken_directed"], "gpu_seconds": t_gpu,
              "oracle_seconds": t_cpu}
        cp["ok"] = bool(same and eu <= tol and ev <= tol and dphi <= TOL_DAMAGE and
                        st["n_broken_directed"] == ko.size and st["step"] == done)
        ok = ok and cp["ok"]
        rec["checkpoints"].append(cp)
        print(f"  step {done}: broken {kg.size} / {ko.size} (pre-cut {2 * len(wl.precut)}), symmetric difference {symdiff}, "
              f"near-threshold {o.near_total}, relL2(u)={eu:.2e} relL2(v)={ev:.2e} max|dphi|={dphi:.1e}  "
              f"[cuda {t_gpu:.1f} s, oracle {t_cpu:.1f} s]  {'ok' if cp['ok'] else 'MISMATCH'}", flush=True)
    sim.destroy()
    rec["ok"] = ok
    if args.out:
        os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
        with open(args.out, "w") as f:
            json.dump(rec, f, indent=1)
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
