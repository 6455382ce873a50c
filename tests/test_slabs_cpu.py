"""Multi-GPU slab decomposition, host logic on CPU.

The partition + exchange loop of paper_2309_11273_b200/slabs.py is driven here with the CPU oracle as the per-rank
stepper: (a) all slabs in one process in lockstep, (b) one slab per process over a world_size-2 gloo group with
point-to-point send/recv.  Both must reproduce the single-domain oracle on the owned nodes BIT FOR BIT (a local
family is the global family in the same ascending order, so every sum has the same addends in the same order) and
give the identical broken-bond set -- that is the statement "one step on owned + 2-delta halo, then one exchange of
u, is exact" (Eq. 2.1 / 2.2 need theta_j of every j within delta, Eq. 1.6 needs the full family of j; Eq. 1.30 is
decided from u at both ends).
"""
import ctypes as C
import os
import pickle
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


class OracleSlabStepper:
    """the oracle's own pieces in the paper's order (extension, dilatation, force, update; oracle/pd_oracle.c steps
    6-9), with step 10 (break on u^{n+1}) run at the start of the next call, i.e. after the halo rows of u^{n+1}
    have been overwritten by their owners' values"""

    def __init__(self, wl):
        from oracle.pd_oracle import PDOracle
        self.o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                          precut=wl.precut, u0=wl.u0, v0=wl.v0)
        self.pending = False

    def flush(self):
        if self.pending and self.o.s_c > 0.0:
            self.o.break_bonds()
        self.pending = False

    def step(self, nsteps):
        from oracle import pd_oracle as P
        o = self.o
        for _ in range(nsteps):
            self.flush()
            o.force_density()
            P.lib().pdo_update(C.c_int64(o.n), C.c_int(o.dim), P._p(o.f), P._p(o.flags), P._p(o.value),
                               C.c_double(o.rho_mass), C.c_double(o.dt), C.c_double(o.ramp_time),
                               C.c_int64(o.step_index), P._p(o.u), P._p(o.v))
            o.step_index += 1
            self.pending = True

    def gather_u(self, idx):
        return self.o.u[np.asarray(idx)].copy()

    def scatter_u(self, idx, values):
        self.o.u[np.asarray(idx)] = np.asarray(values)


def _cases():
    from paper_2309_11273_b200 import workloads as W
    return {
        "config2_small": (W.branching2d(nx=60, ny=36, steps=400), 400, 3),      # fracture, cut along x
        "config4_small": (W.block3d(nx=30, ny=7, nz=6), 40, 3),                  # 3-D, jittered, no fracture
        "config5_small": (W.cylinder3d(r_cells=6, l_cells=40, omega=1500.0), 200, 2),   # 3-D fracture, cut along the axis
    }


def _single(wl, nsteps):
    st = OracleSlabStepper(wl)
    st.step(nsteps)
    st.flush()
    return st.o


def _global_broken(part, o):
    i, j = o.bond_pairs(intact=False)
    own = np.zeros(o.n, bool)
    own[part.owned_local] = True
    keep = own[i]
    return set(zip(part.local[i[keep]].tolist(), part.local[j[keep]].tolist()))


def test_partition_invariants():
    from paper_2309_11273_b200 import slabs
    wl = _cases()["config5_small"][0]
    for world in (1, 2, 3, 5):
        parts, axis = slabs.partition(wl.coords, wl.horizon, world, precut=wl.precut)
        assert axis == 2                                             # the cylinder's axis is the longest extent
        owned = np.concatenate([p.local[p.owned_local] for p in parts])
        assert np.array_equal(np.sort(owned), np.arange(wl.n))      # every node owned exactly once
        c = wl.coords[:, axis]
        for p in parts:
            assert np.all(np.diff(p.local) > 0)
            lo, hi = c[p.local[p.owned_local]].min(), c[p.local[p.owned_local]].max()
            inside = np.nonzero((c >= lo - 2 * wl.horizon) & (c <= hi + 2 * wl.horizon))[0]
            assert np.isin(inside, p.local).all()                    # the 2-delta halo is complete
            halo = np.setdiff1d(np.arange(len(p.local)), p.owned_local)
            got = np.concatenate([p.recv[s] for s in sorted(p.recv)]) if p.recv else np.zeros(0, np.int64)
            assert np.array_equal(np.sort(got), halo)                # every halo node is received from its owner
            for s, idx in p.send.items():                            # what I send is what the peer expects, same order
                q = parts[s]
                assert np.array_equal(p.local[idx], q.local[q.recv[p.rank]])
            # pre-cut pairs: exactly those with both ends local
            pre = np.asarray(wl.precut, np.int64)
            both = np.isin(pre[:, 0], p.local) & np.isin(pre[:, 1], p.local)
            assert len(p.precut_local) == int(both.sum())
            assert np.array_equal(p.local[p.precut_local[:, 0]], pre[both, 0])
        if world > 1:
            sizes = [len(p.owned_local) for p in parts]
            assert max(sizes) - min(sizes) <= 2 * 150                # equal counts up to one lattice layer (113 nodes)


def test_lockstep_slabs_reproduce_single_domain():
    from paper_2309_11273_b200 import slabs
    for name, (wl, nsteps, world) in _cases().items():
        ref = _single(wl, nsteps)
        parts, _ = slabs.partition(wl.coords, wl.horizon, world, precut=wl.precut)
        steppers = [OracleSlabStepper(slabs.local_workload(wl, p)) for p in parts]
        slabs.run_lockstep(parts, steppers, nsteps)
        for st in steppers:
            st.flush()
        u = slabs.assemble_owned(parts, [st.o.u for st in steppers], wl.n, wl.dim)
        v = slabs.assemble_owned(parts, [st.o.v for st in steppers], wl.n, wl.dim)
        assert np.array_equal(u, ref.u) and np.array_equal(v, ref.v), name
        phi = slabs.assemble_owned(parts, [st.o.damage() for st in steppers], wl.n, 0)
        assert np.array_equal(phi, ref.damage()), name
        broken = set().union(*[_global_broken(p, st.o) for p, st in zip(parts, steppers)])
        assert broken == ref.broken_set(), name
        if wl.s_c > 0:
            assert len(broken) > 2 * len(wl.precut), name          # bonds did break during the run


def _gloo_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2309_11273_b200 import slabs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.set_num_threads(1)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl, nsteps, _ = _cases()["config2_small"]
    parts, _ = slabs.partition(wl.coords, wl.horizon, world, precut=wl.precut)
    p = parts[rank]
    st = OracleSlabStepper(slabs.local_workload(wl, p))
    tr = slabs.TorchDistTransport({s: (len(idx), wl.dim) for s, idx in p.recv.items()})
    slabs.SlabRunner(p, st, tr).step(nsteps)
    st.flush()
    dist.barrier()
    with open(f"{out}.{rank}", "wb") as f:
        pickle.dump({"u": st.o.u, "v": st.o.v, "broken": _global_broken(p, st.o)}, f)
    dist.destroy_process_group()


def test_gloo_world2_slabs_reproduce_single_domain(tmp_path):
    from paper_2309_11273_b200 import slabs
    out = str(tmp_path / "s")
    mp.spawn(_gloo_worker, args=(2, 29741, out), nprocs=2, join=True)
    wl, nsteps, _ = _cases()["config2_small"]
    ref = _single(wl, nsteps)
    parts, _ = slabs.partition(wl.coords, wl.horizon, 2, precut=wl.precut)
    res = [pickle.load(open(f"{out}.{r}", "rb")) for r in range(2)]
    u = slabs.assemble_owned(parts, [r["u"] for r in res], wl.n, wl.dim)
    v = slabs.assemble_owned(parts, [r["v"] for r in res], wl.n, wl.dim)
    assert np.array_equal(u, ref.u) and np.array_equal(v, ref.v)
    assert res[0]["broken"] | res[1]["broken"] == ref.broken_set()
    assert len(ref.broken_set()) > 2 * len(wl.precut)
