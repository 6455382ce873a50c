"""GPU parity of the slab decomposition: several pd handles on ONE GPU, each holding one
slab + its 2-delta halo, advanced in lockstep with pd_gather_u / pd_scatter_u as the halo pack / unpack (no rank
waits on another: all kernels of a phase are enqueued on one stream), against the SINGLE-DOMAIN CPU oracle.
Gates as in test_gpu_parity.py: relative L2 of u, v <= 1e-10, identical broken-bond sets, damage to 1e-12."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _cases():
    from paper_2309_11273_b200 import workloads as W
    return {
        "config2_small": (W.branching2d(nx=100, ny=44, steps=600), 600, 3),
        "config4_small": (W.block3d(nx=60, ny=13, nz=11), 120, 2),
        "config5_small": (W.cylinder3d(r_cells=9, l_cells=60, omega=400.0), 300, 3),
    }


def _rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a)


def _broken_owned(part, sim):
    rp, col, intact = sim.get_bond_mask()
    i = np.repeat(np.arange(sim.n), np.diff(rp))
    own = np.zeros(sim.n, bool)
    own[part.owned_local] = True
    keep = own[i] & (intact == 0)
    return set(zip(part.local[i[keep]].tolist(), part.local[col[keep]].tolist()))


@pytest.mark.parametrize("name", ["config2_small", "config4_small", "config5_small"])
def test_slabs_on_one_gpu_match_single_domain_oracle(name):
    from oracle.pd_oracle import PDOracle
    from paper_2309_11273_b200 import pd, slabs
    wl, nsteps, world = _cases()[name]
    o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                 precut=wl.precut, u0=wl.u0, v0=wl.v0)
    parts, _ = slabs.partition(wl.coords, wl.horizon, world, precut=wl.precut)
    sims = [pd.Sim.from_workload(slabs.local_workload(wl, p)) for p in parts]
    done = 0
    for chunk in (1, nsteps // 2, nsteps - 1 - nsteps // 2):
        slabs.run_lockstep(parts, sims, chunk)
        o.step(chunk)
        done += chunk
        u = slabs.assemble_owned(parts, [s.get_u() for s in sims], wl.n, wl.dim)
        v = slabs.assemble_owned(parts, [s.get_v() for s in sims], wl.n, wl.dim)
        if wl.s_c == 0:
            assert _rel(u, o.u) <= TOL and _rel(v, o.v) <= TOL, (name, done)
        else:
            broken = set().union(*[_broken_owned(p, s) for p, s in zip(parts, sims)])
            assert broken == o.broken_set(), (name, done)
            assert _rel(u, o.u) <= 1e-9 and _rel(v, o.v) <= 1e-9, (name, done)   # fracture trajectories
    assert o.near_total == 0
    phi = slabs.assemble_owned(parts, [s.get_damage() for s in sims], wl.n, 0)
    assert np.allclose(phi, o.damage(), rtol=0, atol=1e-12)
    if wl.s_c > 0:
        assert len(o.broken_set()) > 2 * len(wl.precut)
    for s in sims:
        s.destroy()


def test_gather_scatter_roundtrip_and_errors():
    from paper_2309_11273_b200 import pd, workloads as W
    import torch
    wl = W.block3d(nx=20, ny=9, nz=8)
    sim = pd.Sim.from_workload(wl)
    idx = np.random.default_rng(5).permutation(wl.n)[:777].astype(np.int32)
    g = sim.gather_u(idx)
    assert np.array_equal(g.cpu().numpy(), sim.get_u()[idx])
    new = torch.arange(777 * 3, dtype=torch.float64, device=g.device).reshape(777, 3) * 1e-9
    sim.scatter_u(idx, new)
    u = sim.get_u()
    assert np.array_equal(u[idx], new.cpu().numpy())
    rest = np.setdiff1d(np.arange(wl.n), idx)
    assert np.array_equal(u[rest], np.where((wl.flags[rest, None] & (1 << np.arange(3))) != 0, 0.0, wl.u0[rest]))
    assert sim.lib.pd_gather_u(sim.h, None, 5, None) == pd.PD_ERR_ARG
    assert sim.lib.pd_scatter_u(sim.h, None, 0, None) == pd.PD_OK
    sim.destroy()
