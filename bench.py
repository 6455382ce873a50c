#!/usr/bin/env python
"""bench.py -- headline measurement of the OSB-PD explicit step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config5|config5p|config4|config3|config2|config1]
    python bench.py --workload all [--out profiles/r02_configs.json]   # the per-config table of DESIGN.md 5
    python bench.py --impl reference ...      # the CPU oracle as it stands, on the host cores

A "step" is one pass of the whole hot path (dilatation(+break) kernel, force+update kernel: 2 launches)
over the workload.  Metric (BASELINE.json): node-steps/s, FP64; bond-updates/s and the HBM roofline of
the dominant kernel are in the same JSON line.  Default workload = config 5 (3D notched cylinder,
3.144 M nodes, the config the >=60 %-of-HBM-roofline target is quoted on), default step count = the
workload's STATED step count (W warm-up steps + K timed steps = 2000 for config 5), so the timed window
holds the fracture phase of the run (state.broken_directed is printed at the start and at the end).

Timing protocol: pass 1 advances a fresh handle W steps untimed, then exactly K steps between two CUDA
events on the stream the kernels are launched on (-> value, ms_per_step).  Pass 2 repeats the same W + K
steps on a second fresh handle with CUDA events around every launch (-> per-kernel durations over the same
K steps -> roofline).  Inputs are larger than L2 for configs 4, 5, 5' (no flush needed); configs 1-3 fit L2
and say so.

N > 1 (torchrun, one rank per GPU): the path is not sharded ("replicas only"), every
rank advances an independent replica of the workload; value = N * nodes * K / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "node-steps/s"
ALL = ["config1", "config2", "config3", "config4", "config5p", "config5"]
FP64_PEAK = 148 * 64 * 1.965e9   # FP64 lanes x SMs x max SM clock: warp-wide FP64 instructions retire at 2 per clock and SM


def make_workload(name):
    from paper_2309_11273_b200 import workloads as W
    return W.CONFIGS[name]()


def byte_model(n, z, dim, fracture):
    """Algorithmic bytes per launch (fused minimum B2): per directed bond and pass
    4 B index + 1/8 B mask; per node 16d+28 B (dilatation pass) and 40d+29 B (force+update pass)."""
    dil = 4.125 * z + n * (16 * dim + 28 + (8 if fracture else 0))
    frc = 4.125 * z + n * (40 * dim + 29)
    return dil, frc


# FP64 instructions the arithmetic of the shipped kernels needs per directed bond (dilatation, force), by layout
# (counted in the SASS of the FAST step: profiles/r02_kernels.md)
FP64_PER_BOND = {3: (686.0 / 122.0, 1334.0 / 122.0), 2: (7.0, 12.5), 1: (10.0, 22.0), 0: (10.0, 22.0)}
FP64_PER_BOND_2D = {3: (116.0 / 28.0, 244.0 / 28.0)}   # compiled-in 28-offset stencil: 3 / 5 and 7 / 10 per bond


def kernel_source_hash():
    """sha256 over the CUDA sources of the step path (csrc/*.cu, *.cuh): ncu traffic figures are only quoted for the
    build they were captured on.  csrc/aux/ (read-back through static scratch, issue-rate probes) holds separately
    compiled translation units that no step kernel includes or calls and is not part of it."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2309_11273_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


class ClockSampler(threading.Thread):
    """samples nvidia-smi clocks / throttle reasons while the timed region runs"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag, self.proc = index, [], False, None

    def run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append((time.time(), [c.strip() for c in line.split(",")]))
                if self.stop_flag:
                    break
        except Exception:
            pass

    def stop(self):
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()

    def summary(self, t0, t1):
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows]
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": len(rows)}
        try:
            sm = sorted(float(r[0]) for r in rows)
            out["sm_mhz"] = sm[len(sm) // 2]
            out["sm_max_mhz"] = float(rows[0][1])
            out["power_w_max"] = max(float(r[2]) for r in rows)
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            out["reasons"] = [nm for k, nm in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        except Exception:
            pass
        return out


def oracle_sample(wl_name):
    """bounded sample of the benchmark workload for the CPU oracle: same cross-section / lattice,
    material, dt, boundary recipe; fewer nodes and steps (about 10-30 s of CPU work)."""
    from paper_2309_11273_b200 import workloads as W
    if wl_name in ("config5", "config5p"):
        return W.cylinder3d(r_cells=50, l_cells=16), "SAMPLE of the workload: r=50 cells (full cross-section), L=16 cells = 125 760 nodes"
    if wl_name == "config4":
        return W.block3d(nx=80, ny=40, nz=40), "SAMPLE of the workload: 80x40x40 = 128 000 nodes"
    return W.CONFIGS[wl_name](), "full workload"


def time_oracle(wl, steps):
    from oracle import pd_oracle
    o = pd_oracle.PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                           precut=wl.precut, u0=wl.u0, v0=wl.v0)
    t = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t
    return wl.n * steps / dt, dt, o.Z, pd_oracle.num_threads()


def oracle_single_thread(wl_name, steps):
    """node-steps/s of the oracle on ONE host core (SURVEY 8(d) "oracle timing (i)"): a child process with
    OMP_NUM_THREADS=1 (the thread count of an OpenMP runtime is fixed when the library is loaded)"""
    code = ("import json,sys; sys.path.insert(0, %r); import bench; wl, _ = bench.oracle_sample(%r); "
            "v, dt, z, c = bench.time_oracle(wl, %d); print(json.dumps({'value': v, 'seconds': dt, 'cores': c}))"
            % (ROOT, wl_name, steps))
    try:
        out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True,
                             text=True, timeout=600)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception:
        return None


def run_reference(args):
    from paper_2309_11273_b200 import replicas
    if replicas.rank_info()[0] != 0:   # under torchrun rank 0 alone runs and prints the reference arm
        return 0
    name = "config5" if args.workload == "all" else args.workload
    wl, desc = oracle_sample(name)
    k = args.steps if args.steps else 50
    per_step = max(1, min(k, 50 if wl.dim == 3 else 500))
    time_oracle(wl, max(1, min(args.warmup, 1)))          # warm-up (page in, build the .so)
    val, dt, z, cores = time_oracle(wl, per_step)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "node-steps/s", "n_gpus": args.gpus,
        "steps": per_step, "warmup": 1, "ms_per_step": 1e3 * dt / per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{name}:{wl.name}", "sample": desc, "nodes": wl.n, "directed_bonds": z},
        "bond_updates_per_s": z * per_step / dt,
        "cpu_baseline": {"value": val, "unit": "node-steps/s", "cores": cores, "kind": "oracle",
                         "sample": f"{desc}, {per_step} steps"},
        "e2e": {"value": val, "unit": "node-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


def measure(name, K, Wm, local, world, want_e2e, want_cpu):
    """one workload on this rank -> the JSON line (rank 0) or None"""
    import torch
    import torch.distributed as dist
    from paper_2309_11273_b200 import pd, replicas
    rank = replicas.rank_info()[0]
    wl = make_workload(name)
    if K is None:
        K = max(1, wl.steps - Wm)       # W + K = the workload's stated step count
    fracture = wl.s_c > 0

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- pass 1: W warm-up steps, then exactly K steps between CUDA events ----
    t0 = time.perf_counter()
    sim = pd.Sim.from_workload(wl, device=f"cuda:{local}")
    torch.cuda.synchronize()
    t_build = time.perf_counter() - t0
    lay = sim.get_layout()
    n, z = lay["n"], lay["n_directed_bonds"]
    sim.step(Wm)
    broken0 = sim.get_stats()["n_broken_directed"]
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    l0 = sim.get_layout()["step_launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    tw0 = time.time()
    ev0.record()
    sim.step(K)
    ev1.record()
    barrier()
    tw1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = sim.get_layout()["step_launches"] - l0
    sampler.stop()
    clocks = sampler.summary(tw0, tw1)
    ms = replicas.max_over_ranks(ms, device="cuda")
    stats = sim.get_stats()
    u_max = float(np.abs(sim.get_u()).max()) if rank == 0 else 0.0
    sim.destroy()
    # ---- pass 2: the same W + K steps with CUDA events around every launch: per-kernel durations ----
    sim = pd.Sim.from_workload(wl, device=f"cuda:{local}")
    sim.step(Wm)
    kd, kf = sim.step_timed(K)
    sim.destroy()

    # ---- end-to-end through the C-ABI with HOST buffers: the whole job as a user runs it, all of it timed ----
    # pd_create from host arrays (H2D of every input, family build) + the workload's STATED step count + read-back of
    # u, v, damage to host.  The explicit scheme has no per-step input, so the copies are those of the job divided by its
    # steps.  `at_k_steps` is the same sequence with only the K steps of the timed window (pd_create then dominates).
    e2e = None
    if want_e2e:
        def pinned(a):   # page-locked host memory, as the contract says (empty arrays stay as they are)
            a = np.ascontiguousarray(a)
            return torch.from_numpy(a).pin_memory() if a.size else a

        host = {k: pinned(getattr(wl, k)) for k in ("coords", "volumes", "flags", "value", "precut", "u0", "v0")}
        h2d = sum(int(np.prod(a.shape)) * (a.element_size() if hasattr(a, "element_size") else a.itemsize) for a in host.values())
        outs = (torch.empty((wl.n, wl.dim), dtype=torch.float64).pin_memory(), torch.empty((wl.n, wl.dim), dtype=torch.float64).pin_memory(),
                torch.empty(wl.n, dtype=torch.float64).pin_memory())

        def job(steps):
            barrier()
            t0 = time.perf_counter()
            sim2 = pd.Sim(host["coords"], host["volumes"], wl.horizon, **wl.material_kwargs(), flags=host["flags"],
                          value=host["value"], precut=host["precut"], u0=host["u0"], v0=host["v0"], device=f"cuda:{local}")
            sim2.step(steps)
            uo, vo, do = sim2.get_u(outs[0]), sim2.get_v(outs[1]), sim2.get_damage(outs[2])
            barrier()
            te = time.perf_counter() - t0
            d2h = sum(t.numel() * t.element_size() for t in (uo, vo, do))
            sim2.destroy()
            te = replicas.max_over_ranks(te, device="cuda")
            return {"value": replicas.whole_job_throughput(n, steps, te * 1e3, world), "unit": "node-steps/s",
                    "h2d_bytes_per_step": h2d / steps, "d2h_bytes_per_step": d2h / steps, "steps": steps, "seconds": te}

        e2e = job(wl.steps)
        e2e["note"] = ("the whole job: pd_create from pinned host arrays (family build included) + pd_step(stated step count "
                       "of the workload) + pd_get_u/v/damage into pinned host arrays")
        if K != wl.steps:
            e2e["at_k_steps"] = job(K)
    if rank != 0:
        return None

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_kind = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    b_dil, b_frc = byte_model(n, z, wl.dim, fracture)
    # DRAM bytes per launch from the committed ncu capture -- only if it was taken on exactly this kernel source
    traffic, traffic_note = {}, "no ncu capture for this workload"
    try:
        tj = json.load(open(os.path.join(ROOT, "profiles", "r02_traffic.json")))
        if tj.get("kernel_source_sha") != kernel_source_hash():
            traffic_note = "stale: the ncu capture in profiles/r02_traffic.json is of another build of the kernels"
        elif lay.get("layout") != tj.get("layout", {}).get(name):
            traffic_note = "the ncu capture is of another layout"
        else:
            traffic, traffic_note = tj.get(name, {}), tj.get("unit", "")
    except Exception:
        pass
    t_dil, t_frc = kd / K * 1e-3, kf / K * 1e-3
    try:
        fp64_measured = pd.measure_fp64_rate(5)
    except Exception:
        fp64_measured = float("nan")
    dom = ("k_force_update", b_frc, t_frc) if t_frc >= t_dil else ("k_dilatation", b_dil, t_dil)
    achieved = dom[1] / dom[2] / 1e9
    step_s = ms * 1e-3 / K
    fp_d, fp_f = FP64_PER_BOND.get(lay.get("layout"), (10.0, 22.0))
    if wl.dim == 2:
        fp_d, fp_f = FP64_PER_BOND_2D.get(lay.get("layout"), (fp_d, fp_f))
    l2 = 4 * z > 2 * 126e6
    tr = traffic.get(dom[0])
    line = {
        "metric": METRIC, "value": replicas.whole_job_throughput(n, K, ms, world), "unit": "node-steps/s", "n_gpus": world, "steps": K,
        "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{name}:{wl.name}", "nodes": n, "directed_bonds": z, "dim": wl.dim,
                   "fracture": bool(fracture), "stated_steps": wl.steps, "horizon_over_dx": 3.015,
                   "l2": "inputs larger than L2 (no flush needed)" if l2 else "working set fits L2: HBM fraction not meaningful",
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "build_seconds": t_build, "layout": lay},
        "bond_updates_per_s": replicas.whole_job_throughput(z, K, ms, world),
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": dom[0], "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": tr, "traffic_note": traffic_note,
                     "actual_dram_GBps": (tr / dom[2] / 1e9) if tr else None, "peak_kind": peak_kind,
                     "algorithmic_bytes_per_launch": dom[1], "kernel_ms": dom[2] * 1e3,
                     "kernel_ms_is": "mean over the K timed steps, CUDA events around every launch (pass 2)"},
        "kernels": {"k_dilatation": {"ms": t_dil * 1e3, "algorithmic_bytes": b_dil, "GBps": b_dil / t_dil / 1e9},
                    "k_force_update": {"ms": t_frc * 1e3, "algorithmic_bytes": b_frc, "GBps": b_frc / t_frc / 1e9}},
        # co-limiter: FP64 instructions the arithmetic of the shipped kernels needs per directed bond
        "fp64_roofline": {"bound": "alu", "kernel": dom[0], "fp64_per_bond": {"k_dilatation": fp_d, "k_force_update": fp_f},
                          "achieved": (fp_f if dom[0] == "k_force_update" else fp_d) * z / dom[2] / 1e12,
                          "peak": FP64_PEAK / 1e12, "unit": "T FP64 instr/s",
                          "peak_kind": "derived: 148 SM x 64 FP64 lanes x 1.965 GHz (DESIGN.md 5)",
                          "peak_measured": fp64_measured / 1e12,
                          "peak_measured_is": "pd_measure_fp64_rate: 8 independent DFMA chains per thread, 32 warps per SM, best of 5",
                          "frac": (fp_f if dom[0] == "k_force_update" else fp_d) * z / dom[2] / FP64_PEAK,
                          "step_frac": (fp_d + fp_f) * z / step_s / FP64_PEAK},
        "step_roofline": {"algorithmic_bytes_per_step_B2": b_dil + b_frc, "achieved_GBps": (b_dil + b_frc) / step_s / 1e9,
                          "frac_of_peak": (b_dil + b_frc) / step_s / 1e9 / peak, "frac_of_8TBps_nominal":
                          (b_dil + b_frc) / step_s / 8e12},
        "state": {"broken_directed_at_start_of_timed_window": broken0, "broken_directed": stats["n_broken_directed"],
                  "max_damage": stats["max_damage"], "nodes_damage_ge_half": stats["n_nodes_damage_ge_half"],
                  "step": stats["step"], "max_abs_u": u_max},
    }
    if e2e:
        line["e2e"] = e2e
    if want_cpu:
        swl, desc = oracle_sample(name)
        osteps = 600 if swl.dim == 3 else 4000   # about 10-20 s of CPU work
        val, dt, zz, cores = time_oracle(swl, osteps)
        line["cpu_baseline"] = {"value": val, "unit": "node-steps/s", "cores": cores, "kind": "oracle",
                                "sample": f"{desc}, {osteps} steps, {dt:.1f} s"}
        one = oracle_single_thread(name, 40 if swl.dim == 3 else 400)
        if one:
            line["cpu_baseline"]["single_thread"] = {"value": one["value"], "cores": one["cores"], "seconds": one["seconds"]}
    return line


def measure_matrix(name, K, Wm, local):
    """the paper's own 4-SpMV scheme (pd_matrix_*, App. B) on this GPU, on the workload with fracture switched off
    (App. B has no failure step), beside the matrix-free path on the same input: the on-box comparison of DESIGN.md 6"""
    import dataclasses
    import torch
    from paper_2309_11273_b200 import pd
    wl = dataclasses.replace(make_workload(name), s_c=0.0, precut=np.zeros((0, 2), np.int32))
    K = K or 100
    res = {}
    sim = pd.Sim.from_workload(wl, device=f"cuda:{local}")
    n, z = sim.n, sim.get_layout()["n_directed_bonds"]
    t0 = time.perf_counter()
    ms_ = pd.MatrixScheme.from_workload(sim, wl)
    torch.cuda.synchronize()
    t_asm = time.perf_counter() - t0
    for label, obj in (("matrix_free", sim), ("matrix_scheme", ms_)):
        obj.step(Wm)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); obj.step(K); e1.record(); torch.cuda.synchronize()
        res[label] = e0.elapsed_time(e1) / K
    u, v, info = ms_.get()
    err = float(np.linalg.norm(u - sim.get_u()) / max(np.linalg.norm(u), 1e-300))
    ms_.destroy(); sim.destroy()
    # bytes the scheme streams per step: every matrix entry (8 B value + 4 B column) once, the row pointers, the vectors
    nnz = info["nnz_CE"] + info["nnz_CTH"] + info["nnz_KTH"] + info["nnz_KE"]
    vec = 8 * (2 * info["n_bonds"] * 2 + n * (1 + 7 * wl.dim))
    bytes_step = info["matrix_bytes"] + vec
    t = res["matrix_scheme"] * 1e-3
    return {"scheme": "matrix (App. B: 4 CSR SpMV + update, hand-written FP64 kernels)", "metric": METRIC, "unit": "node-steps/s",
            "value": n / t, "ms_per_step": res["matrix_scheme"], "steps": K, "warmup": Wm, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{name}:{wl.name} (fracture off)", "nodes": n, "directed_bonds": z, "undirected_bonds": info["n_bonds"],
                       "nnz": {k: info[k] for k in ("nnz_CE", "nnz_CTH", "nnz_KTH", "nnz_KE")}, "matrix_bytes": info["matrix_bytes"],
                       "assembly_seconds": t_asm},
            "bytes_per_step": bytes_step, "bytes_per_directed_bond_step": bytes_step / z, "achieved_GBps": bytes_step / t / 1e9,
            "matrix_free_ms_per_step": res["matrix_free"], "speedup_matrix_free_over_matrix": res["matrix_scheme"] / res["matrix_free"],
            "relL2_u_matrix_vs_matrix_free": err}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps K (default: stated steps of the workload - warmup)")
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5")
    ap.add_argument("--out", default=None, help="--workload all: write the per-config records to this JSON file")
    ap.add_argument("--scheme", default="matrix-free", choices=["matrix-free", "matrix"],
                    help="matrix: time the paper's own 4-SpMV scheme on this GPU beside the matrix-free path (fracture off)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2309_11273_b200 import replicas
    rank, local, world = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    Wm = max(args.warmup, 3)

    if args.scheme == "matrix":
        if rank == 0:
            print(json.dumps(measure_matrix("config4" if args.workload == "all" else args.workload, args.steps, Wm, local)))
        if world > 1:
            dist.destroy_process_group()
        return 0
    if args.workload == "all":
        recs = []
        for name in ALL:
            line = measure(name, args.steps, Wm, local, world, False, False)
            if line:
                recs.append(line)
        if rank == 0:
            out = {"kernel_source_sha": kernel_source_hash(), "records": recs}
            if args.out:
                with open(args.out, "w") as f:
                    json.dump(out, f, indent=1)
            print(json.dumps({"metric": METRIC, "workload": "all", "records": [
                {"workload": r["config"]["workload"], "ms_per_step": r["ms_per_step"], "value": r["value"]} for r in recs]}))
    else:
        line = measure(args.workload, args.steps, Wm, local, world, not args.no_e2e, not args.no_cpu_baseline)
        if line:
            print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
