"""pd_get_u_static (include/pd.h): the read-back of u^n that allocates no device memory, against pd_get_u.

Collected last on purpose (the run is `pytest -x`): the static scratch array is shared by every call in the
process, so this file also runs after all other GPU tests have used the library, and must pass alone in a fresh
process as well.

Both entry points copy the same stored doubles, so the outputs must be IDENTICAL bit for bit; the relative-L2 bound
of the parity tests (TOL = 1e-10, tests/test_gpu_parity.py) is asserted beside it.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10

_ENV_KEYS = ("PD_LAT_UNIFORM", "PD_FORCE_GENERIC", "PD_BALL", "PD_DISC", "PD_GRAPH")


def _rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a)


def _same(a, b):
    assert _rel(a, b) <= TOL
    assert np.array_equal(a, b)


def _cases():
    from paper_2309_11273_b200 import workloads as W
    return {
        # storage of u^n                                        expected layout code (pd_get_layout)
        "uniform3d": (W.cylinder3d(r_cells=9, l_cells=34, omega=400.0), {}, 3),     # {u_0, u_1} + u_2 arrays, fracture
        "uniform2d": (W.cantilever2d(nx=50, ny=10), {}, 3),                         # {u_0, u_1} array, shuffled node order
        "lattice_records": (W.block3d(nx=37, ny=13, nz=11), {}, 1),                 # records of the dense lattice, ragged n
        "sliced_ell": (W.block3d(nx=14, ny=9, nz=8), {"PD_FORCE_GENERIC": "1"}, 0),  # AoSoA-32 neighbour records
    }


@pytest.mark.parametrize("name", ["uniform3d", "uniform2d", "lattice_records", "sliced_ell"])
def test_static_scratch_read_matches_get_u_twice_in_a_row(name, monkeypatch):
    from paper_2309_11273_b200 import pd
    wl, env, code = _cases()[name]
    for k in _ENV_KEYS:
        monkeypatch.delenv(k, raising=False)
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    sim = pd.Sim.from_workload(wl)
    assert sim.get_layout()["layout"] == code
    assert wl.n * wl.dim <= pd.STATIC_MAX_DOUBLES
    _same(sim.get_u_static(), sim.get_u())       # before any step: the initial condition
    sim.step(40)
    ref = sim.get_u()
    a = sim.get_u_static()
    b = sim.get_u_static()                       # two calls in a row share the scratch
    _same(a, ref)
    _same(b, ref)
    sim.step(7)                                  # odd step count: the other u buffer is current now
    ref2 = sim.get_u()
    assert not np.array_equal(ref2, ref)
    _same(sim.get_u_static(), ref2)
    _same(sim.get_u_static(), ref2)
    sim.destroy()


def test_static_scratch_read_allocates_nothing_and_takes_device_pointers():
    """with the handle's allocator failing every request, pd_get_u cannot stage its copy (PD_ERR_ALLOC); the static
    entry point still answers, into host memory and into a caller-owned device buffer, and holds no extra memory"""
    import torch
    from paper_2309_11273_b200 import pd, workloads as W
    wl = W.cylinder3d(r_cells=9, l_cells=34, omega=400.0)
    sim = pd.Sim.from_workload(wl)
    sim.step(25)
    ref = sim.get_u()
    held = sim.get_layout()["device_bytes"]
    live = len(sim._rt.live)
    sim._rt.fail_allocs = True
    with pytest.raises(pd.PdError) as ei:
        sim.get_u()
    assert ei.value.code == pd.PD_ERR_ALLOC
    _same(sim.get_u_static(), ref)
    out = torch.full((wl.n, wl.dim), float("nan"), dtype=torch.float64, device="cuda:0")
    sim.get_u_static(out)
    _same(out.cpu().numpy(), ref)
    sim._rt.fail_allocs = False
    assert sim.get_layout()["device_bytes"] == held and len(sim._rt.live) == live
    sim.destroy()


def test_static_scratch_is_shared_and_stale_contents_are_never_returned():
    """a large read followed by a smaller one of another handle: the second sees only its own dim*n doubles"""
    from paper_2309_11273_b200 import pd, workloads as W
    big = pd.Sim.from_workload(W.block3d(nx=37, ny=13, nz=11))
    small = pd.Sim.from_workload(W.cantilever2d(nx=40, ny=10))
    big.step(10); small.step(10)
    rb, rs = big.get_u(), small.get_u()
    _same(big.get_u_static(), rb)
    _same(small.get_u_static(), rs)
    _same(big.get_u_static(), rb)
    _same(small.get_u_static(), rs)
    big.destroy(); small.destroy()


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    """dim*n > PD_STATIC_MAX_DOUBLES: PD_ERR_LIMIT with a message that names the limit, nothing written, handle intact"""
    from paper_2309_11273_b200 import pd, workloads as W
    wl = W.cantilever2d(nx=1025, ny=512)          # 2 x 524800 = 1049600 > 1048576
    assert wl.n * wl.dim > pd.STATIC_MAX_DOUBLES
    sim = pd.Sim.from_workload(wl)
    sim.step(3)
    out = np.full((wl.n, wl.dim), -7.0)
    with pytest.raises(pd.PdError) as ei:
        sim.get_u_static(out)
    assert ei.value.code == pd.PD_ERR_LIMIT
    assert "PD_STATIC_MAX_DOUBLES" in str(ei.value) and str(pd.STATIC_MAX_DOUBLES) in str(ei.value)
    assert np.all(out == -7.0)
    ref = sim.get_u()                             # the allocating path still serves the handle
    assert np.isfinite(ref).all() and np.linalg.norm(ref) > 0
    sim.destroy()
    # right at the limit the call is served: 2 x 524288 = 1048576
    wl = W.cantilever2d(nx=1024, ny=512)
    assert wl.n * wl.dim == pd.STATIC_MAX_DOUBLES
    sim = pd.Sim.from_workload(wl)
    sim.step(3)
    _same(sim.get_u_static(), sim.get_u())
    sim.destroy()
