"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances (north star / DESIGN.md):
  no-fracture configs : relative L2 of u and of v <= 1e-10 after the stated steps
  fracture configs    : identical broken-bond sets, except bonds whose stretch is within
                        1e-9 relative of s_c at the step they break (counted, must be zero here
                        unless reported)
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10

# the code paths of the library: the layout is chosen inside pd_create; the environment
# switches exist for exactly this purpose (and for profiling).  Layout codes (pd_get_layout): 3 = uniform lattice with
# the stencil of horizon 3.015 dx compiled in (122 offsets in 3-D, 28 in 2-D: configs 1, 2, 3, 5), 2 = uniform
# lattice (constant bond geometry per stencil offset, table-driven kernels: any other stencil),
# 1 = dense lattice with per-bond geometry (jittered config 4; PD_LAT_UNIFORM=0 forces it), 0 = sliced ELL.
LAYOUTS = {
    "default": ({}, None),
    # uniform lattice, records through L1 instead of TMA-staged planes; rows per lane swapped (2 in 3-D, 4 in 2-D);
    # plain launches instead of CUDA graphs
    # (PD_BALL=0, PD_DISC=0: the table-driven kernels also where the stencil is the compiled-in 122-offset ball of
    # pd_lattice_ball.cu / the 28-offset disc of pd_lattice_disc.cu)
    "uniform_direct": ({"PD_ULAT_STAGED": "0", "PD_ULAT_DIL_ROWS": "-1", "PD_ULAT_FRC_ROWS": "-1", "PD_GRAPH": "0",
                        "PD_BALL": "0", "PD_DISC": "0"}, None),
    # staged planes with 3 buffers in flight, rows per lane swapped, 2 row groups per CTA
    "uniform_nb3": ({"PD_ULAT_NB": "3", "PD_ULAT_DIL_ROWS": "-1", "PD_ULAT_FRC_ROWS": "-1", "PD_ULAT_DIL_CY": "2",
                     "PD_ULAT_FRC_CY": "2", "PD_BALL": "0", "PD_DISC": "0"}, None),
    # table-driven staged kernels with their default shape
    "uniform_table": ({"PD_BALL": "0", "PD_DISC": "0"}, None),
    # compiled-in stencil kernels in their other launch shape: 4 rows per CTA, 3 plane buffers in flight
    "ball_cy4_nb3": ({"PD_BALL_CY": "4", "PD_BALL_NB": "3"}, None),
    "lattice_general": ({"PD_LAT_UNIFORM": "0"}, 1),
    "lattice_general_2rows": ({"PD_LAT_UNIFORM": "0", "PD_DIR_DIL_ROWS": "2", "PD_DIR_FRC_ROWS": "2"}, 1),
    "sliced_ell": ({"PD_FORCE_GENERIC": "1"}, 0),
}
_ENV_KEYS = ("PD_LAT_UNIFORM", "PD_FORCE_GENERIC", "PD_DIR_DIL_ROWS", "PD_DIR_FRC_ROWS", "PD_ULAT_DIL_ROWS",
             "PD_ULAT_FRC_ROWS", "PD_ULAT_STAGED", "PD_ULAT_NB", "PD_ULAT_DIL_CY", "PD_ULAT_FRC_CY", "PD_GRAPH", "PD_BALL", "PD_BALL_CY", "PD_BALL_NB", "PD_DISC")


@pytest.fixture(params=list(LAYOUTS))
def layout(request, monkeypatch):
    env, code = LAYOUTS[request.param]
    for k in _ENV_KEYS:
        monkeypatch.delenv(k, raising=False)
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    return code


def _expect_layout(code, wl):
    """the layout pd_create must pick by itself: jittered lattices cannot take the uniform path"""
    if code is not None:
        return code
    if wl.name == "block3d" and wl.meta.get("jitter", 1.0) != 0.0:
        return 1
    import os
    # 3: the kernels with the stencil compiled in (122 offsets in 3-D, 28 in 2-D)
    return 3 if os.environ.get("PD_BALL" if wl.dim == 3 else "PD_DISC", "1") != "0" else 2


def _oracle(wl):
    from oracle.pd_oracle import PDOracle
    return PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                    precut=wl.precut, u0=wl.u0, v0=wl.v0)


def _sim(wl, **kw):
    from paper_2309_11273_b200 import pd
    return pd.Sim.from_workload(wl, **kw)


def _rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a)


def _broken_set(sim):
    rp, col, intact = sim.get_bond_mask()
    i = np.repeat(np.arange(sim.n), np.diff(rp))
    return set(zip(i[intact == 0].tolist(), col[intact == 0].tolist())), rp, col


def _small_cases():
    from paper_2309_11273_b200 import workloads as W
    return {
        "config1_full": (W.cantilever2d(), 2000),
        "config2_small": (W.branching2d(nx=100, ny=44, steps=600), 600),
        "config3_small": (W.impact2d(nx=72, ny=72), 500),
        "config4_small": (W.block3d(nx=37, ny=13, nz=11), 120),          # ragged: 5291 nodes, not /32
        "config5_small": (W.cylinder3d(r_cells=9, l_cells=34, omega=400.0), 300),   # omega raised so the short run breaks bonds
        # long enough along the lane axis for row groups with every family complete (the FAST bodies of the
        # compiled-in stencil, their break filter and exact pass), ragged last chunk
        "config5_long": (W.cylinder3d(r_cells=9, l_cells=100, omega=400.0), 300),
        "block3d_uniform": (W.block3d(nx=70, ny=13, nz=11, jitter=0.0), 120),       # unjittered: uniform lattice, no fracture
    }


@pytest.mark.parametrize("name", ["config1_full", "config4_small", "block3d_uniform"])
def test_no_fracture_trajectory(name, layout):
    wl, nsteps = _small_cases()[name]
    sim, o = _sim(wl), _oracle(wl)
    assert sim.get_layout()["layout"] == _expect_layout(layout, wl)
    # pre-processing parity: family sizes, m, theta of the initial field
    rp = sim.get_bond_mask(rows_only=True)
    assert np.array_equal(rp, o.rowptr)
    m, th = sim.get_node_fields()
    assert _rel(m, o.m) <= 1e-14
    assert _rel(th, o.dilatation()) <= 1e-11
    done = 0
    for chunk in (1, 2, nsteps - 3):
        sim.step(chunk); o.step(chunk); done += chunk
        assert _rel(sim.get_u(), o.u) <= TOL, (name, done)
        assert _rel(sim.get_v(), o.v) <= TOL, (name, done)
    assert sim.get_stats()["step"] == nsteps
    assert sim.get_stats()["n_broken_directed"] == 0 and np.all(sim.get_damage() == 0.0)
    sim.destroy()


@pytest.mark.parametrize("name", ["config2_small", "config3_small", "config5_small", "config5_long"])
def test_fracture_broken_sets(name, layout):
    wl, nsteps = _small_cases()[name]
    sim, o = _sim(wl), _oracle(wl)
    assert sim.get_layout()["layout"] == _expect_layout(layout, wl)
    b0, rp, col = _broken_set(sim)
    assert np.array_equal(rp, o.rowptr)
    assert b0 == o.broken_set() and len(b0) == 2 * len(wl.precut)
    assert np.allclose(sim.get_damage(), o.damage(), rtol=0, atol=1e-13)
    total = 0
    for chunk in (nsteps // 4, nsteps // 4, nsteps - 2 * (nsteps // 4)):
        sim.step(chunk)
        total += o.step(chunk)
        bs, _, _ = _broken_set(sim)
        assert o.near_total == 0, "near-threshold events must be reported, none expected here"
        assert bs == o.broken_set(), (name, len(bs), len(o.broken_set()))
        assert np.allclose(sim.get_damage(), o.damage(), rtol=0, atol=1e-12)
    assert total > 0, "the case must actually break bonds"
    st = sim.get_stats()
    assert st["n_broken_directed"] == len(o.broken_set())
    assert st["max_damage"] == pytest.approx(o.phi.max(), abs=1e-12)
    assert st["n_nodes_damage_ge_half"] == int((o.phi >= 0.5).sum())
    # trajectories stay close too (same break history => same linear pieces)
    assert _rel(sim.get_u(), o.u) <= 1e-9 and _rel(sim.get_v(), o.v) <= 1e-9
    sim.destroy()


def test_compiled_in_stencil_run_to_run_reproducible():
    """The break test of the compiled-in stencil kernels goes through a worklist filled with atomics (entry order varies
    from run to run) and clears octant-word bits with atomics: the state must not depend on that order.  Two runs of the
    long cylinder, bonds breaking, must agree bit for bit in u, v, damage and the bond masks."""
    wl, nsteps = _small_cases()["config5_long"]
    out = []
    for _ in range(2):
        sim = _sim(wl)
        assert sim.get_layout()["layout"] == 3
        sim.step(nsteps)
        rp, col, intact = sim.get_bond_mask()
        out.append((sim.get_u().copy(), sim.get_v().copy(), sim.get_damage().copy(), intact.copy()))
        sim.destroy()
    assert int((out[0][3] == 0).sum()) > 2 * len(wl.precut), "the case must break bonds"
    for a, b in zip(out[0], out[1]):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("fracture", [False, True])
def test_uniform_block_traction_ramp_and_mixed_dofs(fracture):
    """Eq. 2.11 with the ramped body force g(t_n) b and per-dof boundary flags (App. B; C-3, C-4, C-14)
    on the compiled-in stencil kernels of a plain 3-D lattice: traction on the far face ramped over 40 steps, the near
    face clamped in x only, one edge with a prescribed z velocity; with and without the break filter / break test
    (s_c chosen so that the loaded face tears off within the run)."""
    from paper_2309_11273_b200 import workloads as W
    wl = W.block3d(nx=70, ny=13, nz=11, jitter=0.0)
    ix = np.rint(wl.coords[:, 0] / wl.dx - 0.5).astype(int)
    iy = np.rint(wl.coords[:, 1] / wl.dx - 0.5).astype(int)
    wl.u0[:] = 0.0
    wl.flags[:] = 0
    wl.value[:] = 0.0
    wl.flags[ix < 3] = W.CLAMP_X
    far = ix >= 69
    wl.flags[far] = W.BODY_FORCE
    wl.value[far, 0] = 4.0e6 / wl.dx            # sigma / dx on the outermost node layer (C-14)
    wl.value[far, 1] = -1.0e6 / wl.dx
    edge = (ix >= 30) & (ix < 40) & (iy == 0)
    wl.flags[edge] |= W.PRESC_Z
    wl.value[edge, 2] = 0.05
    wl.ramp_time = 40 * wl.dt
    if fracture:
        wl.s_c = 2.0e-5
    sim, o = _sim(wl), _oracle(wl)
    assert sim.get_layout()["layout"] == 3
    nsteps, total = 120, 0
    for chunk in (1, 39, 80):
        sim.step(chunk)
        total += o.step(chunk)
        if fracture:
            bs, _, _ = _broken_set(sim)
            assert o.near_total == 0 and bs == o.broken_set()
        assert _rel(sim.get_u(), o.u) <= (1e-9 if fracture else TOL)
        assert _rel(sim.get_v(), o.v) <= (1e-9 if fracture else TOL)
    assert (total > 0) == fracture
    assert sim.get_stats()["step"] == nsteps
    sim.destroy()


def test_nonuniform_volume_and_device_pointers():
    """general path: non-uniform V, inputs/outputs as torch CUDA tensors, library allocator."""
    import torch
    from paper_2309_11273_b200 import pd, workloads as W
    wl = W.block3d(nx=14, ny=9, nz=8)
    rng = np.random.default_rng(11)
    wl.volumes = wl.volumes * rng.uniform(0.7, 1.3, wl.n)
    o = _oracle(wl)
    dev = torch.device("cuda:0")
    sim = pd.Sim(torch.from_numpy(wl.coords).to(dev), torch.from_numpy(wl.volumes).to(dev), wl.horizon,
                 **wl.material_kwargs(), flags=torch.from_numpy(wl.flags).to(dev), u0=torch.from_numpy(wl.u0).to(dev),
                 use_torch_allocator=False)
    assert sim.get_layout()["uniform_volume"] == 0
    sim.step(60); o.step(60)
    out = torch.empty((wl.n, 3), dtype=torch.float64, device=dev)
    sim.get_u(out)
    assert _rel(out.cpu().numpy(), o.u) <= TOL and _rel(sim.get_v(), o.v) <= TOL
    sim.destroy()


def test_edge_cases_and_errors():
    from paper_2309_11273_b200 import pd
    # two nodes, one bond: hand value F1 = 18 kappa a V / r^2 reproduced through one step
    x = np.array([[0, 0, 0], [0.6, 0.0, 0.8]])
    kw = dict(dim=3, mode=0, E=5.0, nu=0.2, rho=2.0, dt=1e-3)
    a = 2e-4
    sim = pd.Sim(x, np.full(2, 0.3), 1.5, **kw, u0=np.array([[0, 0, 0], a * x[1]]))
    sim.step(1)
    kappa = 5.0 / (3 * (1 - 0.4))
    f1 = 18 * kappa * a / 1.0 ** 2 * x[1]                      # force density on node 0 (V cancels: F/V)
    assert np.allclose(sim.get_v()[0], 1e-3 * f1 / 2.0, rtol=1e-12)
    assert np.allclose(sim.get_v()[1], -sim.get_v()[0], rtol=1e-14)
    sim.destroy()
    # isolated node
    with pytest.raises(pd.PdError) as ei:
        pd.Sim(np.array([[0.0, 0], [1, 0], [9, 9]]), np.ones(3), 1.5, dim=2, mode=1, E=1.0, nu=0.2, rho=1.0, dt=1.0)
    assert ei.value.code == pd.PD_ERR_ISOLATED
    # bad arguments
    for bad in (dict(nu=0.5), dict(E=-1.0), dict(dt=0.0), dict(mode=0)):
        k2 = dict(dim=2, mode=1, E=1.0, nu=0.2, rho=1.0, dt=1.0); k2.update(bad)
        with pytest.raises(pd.PdError) as ei:
            pd.Sim(np.array([[0.0, 0], [1, 0]]), np.ones(2), 1.5, **k2)
        assert ei.value.code == pd.PD_ERR_ARG
    # pre-cut pair that is not a bond
    with pytest.raises(pd.PdError) as ei:
        pd.Sim(np.array([[0.0, 0], [1, 0], [2, 0]]), np.ones(3), 1.5, dim=2, mode=1, E=1.0, nu=0.2, rho=1.0, dt=1.0,
               precut=np.array([[0, 2]], np.int32))
    assert ei.value.code == pd.PD_ERR_ARG
    # step(0) is a no-op; empty pre-cut list
    sim = pd.Sim(np.array([[0.0, 0], [1, 0]]), np.ones(2), 1.5, dim=2, mode=2, E=1.0, nu=0.2, rho=1.0, dt=1e-9,
                 precut=np.zeros((0, 2), np.int32))
    sim.step(0)
    assert sim.get_stats()["step"] == 0 and sim.get_stats()["n_directed_bonds"] == 2
    sim.destroy()


def test_threshold_bond(layout):
    """a single bond exactly at the threshold breaks, one ulp below does not (Eq. 1.30 PAPER.md:417-425,
    reading C-7), on every code path and exactly like the oracle.  Both nodes carry a prescribed velocity
    0 on both dofs, so u^1 = u^0 and the failure check of step 1 sees the stretch s = a0 exactly."""
    from paper_2309_11273_b200 import pd
    from oracle.pd_oracle import PDOracle
    s_c = 1e-3
    x = np.array([[0.0, 0.0], [1.0, 0.0]])
    kw = dict(dim=2, mode=2, E=1.0, nu=0.2, rho=1.0, dt=1e-9, s_c=s_c)
    fl = np.array([24, 24], np.uint8)
    for a0, broken in ((s_c, True), (np.nextafter(s_c, 0), False), (np.nextafter(s_c, 1), True), (0.5 * s_c, False),
                       (-2 * s_c, False)):
        u0 = np.array([[0.0, 0.0], [a0, 0.0]])
        o = PDOracle(x, np.ones(2), 1.5, **kw, flags=fl, value=np.zeros((2, 2)), u0=u0)
        o.step(1)
        assert len(o.broken_set()) == (2 if broken else 0)
        sim = pd.Sim(x, np.ones(2), 1.5, **kw, flags=fl, value=np.zeros((2, 2)), u0=u0)
        sim.step(1)
        assert np.array_equal(sim.get_u(), u0)
        assert sim.get_stats()["n_broken_directed"] == (2 if broken else 0), (a0, broken)
        bs, _, _ = _broken_set(sim)
        assert bs == o.broken_set()
        assert np.array_equal(sim.get_damage(), o.damage())
        sim.destroy()


@pytest.mark.parametrize("case", ["cylinder3d", "branching2d_table"])
def test_step_error_is_returned_and_state_kept(case, monkeypatch):
    """a launch that cannot be prepared (device allocation failing inside pd_step) must come back as an error
    code and leave the step counter and the buffers where they were.  (The compiled-in 3-D stencil kernels allocate
    their octant words, tile flags and worklist at the first step, the table-driven kernels their tables; the
    compiled-in 2-D kernels allocate nothing, hence PD_DISC=0 for the 2-D case.)"""
    from paper_2309_11273_b200 import pd, workloads as W
    if case == "cylinder3d":
        wl = W.cylinder3d(r_cells=9, l_cells=34, omega=400.0)
    else:
        monkeypatch.setenv("PD_DISC", "0")
        wl = W.branching2d(nx=40, ny=24)
    o = _oracle(wl)
    sim = _sim(wl)
    sim._rt.fail_allocs = True          # fault injection: the allocator callback returns NULL
    with pytest.raises(pd.PdError) as ei:
        sim.step(3)
    assert ei.value.code == pd.PD_ERR_ALLOC
    sim._rt.fail_allocs = False
    assert sim.get_stats()["step"] == 0
    sim.step(5); o.step(5)
    assert sim.get_stats()["step"] == 5
    assert _rel(sim.get_u(), o.u) <= TOL and _rel(sim.get_v(), o.v) <= TOL
    sim.destroy()


def test_lattice_layout_fallbacks():
    """bodies the dense lattice layout must decline by itself (pd_lattice.cu): a lattice whose stencil has
    more than 128 offsets (horizon 4.1 dx in 3-D: 250+), and a body that fills < 20 % of its bounding
    box.  Both must come back in the sliced-ELL layout and match the oracle."""
    from paper_2309_11273_b200 import pd
    from oracle.pd_oracle import PDOracle
    kw = dict(dim=3, mode=0, E=3.0, nu=0.25, rho=1.5, dt=1e-3)
    g = np.stack(np.meshgrid(np.arange(12), np.arange(9), np.arange(8), indexing="ij"), -1).reshape(-1, 3).astype(float)
    cases = {"wide_stencil": (0.1 * (g + 0.5), 0.41)}
    a = 0.1 * (np.stack(np.meshgrid(np.arange(30), np.arange(4), np.arange(4), indexing="ij"), -1).reshape(-1, 3) + 0.5)
    cases["sparse_box"] = (np.concatenate([a, a + np.array([0.0, 2.0, 2.0])]), 0.3015)   # two bars, 5.5 % of their bounding box
    for name, (x, hor) in cases.items():
        n = len(x)
        u0 = 1e-4 * np.sin(7.0 * x[:, [1, 2, 0]])
        sim = pd.Sim(x, np.full(n, 1e-3), hor, **kw, u0=u0)
        assert sim.get_layout()["layout"] == 0, name
        o = PDOracle(x, np.full(n, 1e-3), hor, **kw, u0=u0)
        assert np.array_equal(sim.get_bond_mask(rows_only=True), o.rowptr)
        sim.step(25); o.step(25)
        assert _rel(sim.get_u(), o.u) <= TOL and _rel(sim.get_v(), o.v) <= TOL, name
        sim.destroy()


def test_point_cloud_general_layout():
    """a random cloud (cells with 0, 1 or several nodes): the sliced-ELL layout with its FLAT segments"""
    from paper_2309_11273_b200 import pd
    from oracle.pd_oracle import PDOracle
    rng = np.random.default_rng(5)
    n = 3000
    x = rng.uniform(0.0, 1.0, (n, 3)) * np.array([1.0, 0.6, 0.4])
    kw = dict(dim=3, mode=0, E=3.0, nu=0.25, rho=1.5, dt=2e-3)
    u0 = 1e-4 * np.sin(3.0 * x[:, [1, 2, 0]])
    sim = pd.Sim(x, np.full(n, 1.0 / n), 0.16, **kw, u0=u0)
    assert sim.get_layout()["layout"] == 0
    o = PDOracle(x, np.full(n, 1.0 / n), 0.16, **kw, flags=None, value=None, precut=None, u0=u0, v0=None)
    assert np.array_equal(sim.get_bond_mask(rows_only=True), o.rowptr)
    sim.step(40); o.step(40)
    assert _rel(sim.get_u(), o.u) <= TOL and _rel(sim.get_v(), o.v) <= TOL
    sim.destroy()


def test_full_size_config5p_sampled():
    """BASELINE-size workload (config 5', 1 257 600 nodes) in the launch configuration bench.py times:
    a few steps against the oracle -- every node for u and v, the complete broken-bond set, damage."""
    from paper_2309_11273_b200 import workloads as W
    wl = W.CONFIGS["config5p"]()
    sim, o = _sim(wl), _oracle(wl)
    assert sim.get_layout()["layout"] == 3   # the compiled-in 122-offset stencil kernels
    assert sim.get_stats()["n_directed_bonds"] == o.Z
    sim.step(3); o.step(3)
    assert _rel(sim.get_u(), o.u) <= TOL and _rel(sim.get_v(), o.v) <= TOL
    st = sim.get_stats()
    assert st["n_broken_directed"] == len(o.broken_set()) == 2 * len(wl.precut)
    rng = np.random.default_rng(0)
    idx = rng.integers(0, wl.n, 2000)
    assert np.allclose(sim.get_damage()[idx], o.damage()[idx], rtol=0, atol=1e-12)
    sim.destroy()


@pytest.mark.parametrize("generic", [False, True])
def test_geometric_extension_variant(generic, monkeypatch):
    """the geometric extension e = ||xi + eta|| - ||xi|| of App. C in the dilatation,
    the force and the failure stretch (pd_material.extension = PD_EXT_GEOMETRIC), against the oracle's variant:
    a FINITE rigid rotation gives zero force, trajectories agree to 1e-10, broken sets are identical."""
    from paper_2309_11273_b200 import pd, workloads as W
    from oracle.pd_oracle import PDOracle
    for k in _ENV_KEYS:
        monkeypatch.delenv(k, raising=False)
    if generic:
        monkeypatch.setenv("PD_FORCE_GENERIC", "1")
    # finite rotation: zero force with the geometric extension (the linearized model pushes back)
    wl = W.block3d(nx=16, ny=9, nz=8)
    x = wl.coords
    c, s_ = np.cos(0.4), np.sin(0.4)
    u0 = x @ np.array([[c, -s_, 0], [s_, c, 0], [0, 0, 1.0]]).T - x
    kw = dict(wl.material_kwargs()); kw["dt"] = 1e-7
    sim = pd.Sim(x, wl.volumes, wl.horizon, **kw, u0=u0, extension="geometric")
    assert sim.get_layout()["layout"] == (0 if generic else 1)
    sim.step(1)
    v_geo = np.abs(sim.get_v()).max()
    sim.destroy()
    sim = pd.Sim(x, wl.volumes, wl.horizon, **kw, u0=u0)
    sim.step(1)
    v_lin = np.abs(sim.get_v()).max()
    sim.destroy()
    assert v_geo <= 1e-9 * v_lin and v_lin > 0
    # trajectories and broken sets
    for wl, nsteps in ((W.block3d(nx=21, ny=10, nz=9), 60), (W.branching2d(nx=80, ny=40, steps=500), 420),
                       (W.cylinder3d(r_cells=8, l_cells=30, omega=400.0), 120)):
        o = PDOracle(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                     precut=wl.precut, u0=wl.u0, v0=wl.v0, extension="geometric")
        sim = pd.Sim.from_workload(wl, extension="geometric")
        assert sim.get_layout()["layout"] == (0 if generic else 1)   # the uniform-lattice path is linearized only
        sim.step(nsteps); o.step(nsteps)
        assert _rel(sim.get_u(), o.u) <= (TOL if wl.s_c == 0 else 1e-9), wl.name
        assert _rel(sim.get_v(), o.v) <= (TOL if wl.s_c == 0 else 1e-9), wl.name
        bs, _, _ = _broken_set(sim)
        assert bs == o.broken_set() and o.near_total == 0, wl.name
        if wl.s_c > 0:
            assert len(bs) > 2 * len(wl.precut), "the case must actually break bonds"
        sim.destroy()


def test_matrix_scheme_matches_oracle():
    """the paper's matrix-based scheme (CE, CTH, KTH, KE of Eqs. 2.7-2.10 + the solver body of App. B,
    PAPER.md:860-885) with hand-written CSR SpMVs, against the oracle (no fracture): relative L2 of u, v <= 1e-10,
    and against the matrix-free path of the same library"""
    from paper_2309_11273_b200 import pd, workloads as W
    for wl, nsteps in ((W.cantilever2d(), 300), (W.block3d(nx=24, ny=11, nz=9), 80)):
        sim, o = _sim(wl), _oracle(wl)
        ms = pd.MatrixScheme.from_workload(sim, wl)
        ms.step(nsteps); sim.step(nsteps); o.step(nsteps)
        u, v, info = ms.get()
        assert info["n_bonds"] * 2 == o.Z and info["nnz_CE"] == 2 * wl.dim * info["n_bonds"] and info["step"] == nsteps
        assert info["nnz_KTH"] == wl.dim * (o.Z + wl.n) and info["nnz_KE"] == wl.dim * o.Z and info["nnz_CTH"] == o.Z
        assert _rel(u, o.u) <= TOL and _rel(v, o.v) <= TOL, wl.name
        assert _rel(u, sim.get_u()) <= TOL
        ms.destroy(); sim.destroy()


@pytest.mark.parametrize("env", [{}, {"PD_LAT_UNIFORM": "0"}, {"PD_FORCE_GENERIC": "1"}])
def test_adr_quasi_static_driver(env, monkeypatch):
    """adaptive dynamic relaxation (pd_adr_step) against the oracle's ADR (oracle/pd_adr.py,
    itself pinned to the direct solve).  The damping estimate c^n divides force differences by velocities that pass
    through zero, so two correct implementations drift apart in their ITERATES after some tens of iterations (measured:
    1e-14 after 8 iterations, 1e-3 after 50 under continuous displacement loading) while converging to the same
    equilibrium; the test therefore checks (a) iterate-by-iterate equality while it holds, on a smooth load for hundreds
    of iterations; (b) a failure check inside the first iterations: identical broken sets; (c) the converged states."""
    from paper_2309_11273_b200 import pd
    from oracle.pd_oracle import PDOracle
    from oracle.pd_adr import ADROracle
    for k in _ENV_KEYS:
        monkeypatch.delenv(k, raising=False)
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    # (a) bar 14 x 6 x 5 cells, one end clamped, body force on the other end layer
    g = np.stack(np.meshgrid(np.arange(14), np.arange(6), np.arange(5), indexing="ij"), -1).reshape(-1, 3)
    x = (g + 0.5) * 1e-3
    fl = np.zeros(len(x), np.uint8); fl[g[:, 0] < 2] = 7; fl[g[:, 0] == 13] |= 64
    val = np.zeros_like(x); val[g[:, 0] == 13] = [3e9, 5e8, 0.0]
    kw = dict(dim=3, mode=0, E=72e9, nu=0.22, rho=1.0, dt=1.0)
    vol = np.full(len(x), 1e-9)
    lam = 0.3 * 72e9 / 1e-6          # >= lambda_max(K)/4 for this lattice (the run stays bounded and converges)
    o = PDOracle(x, vol, 3.015e-3, **kw, flags=fl, value=val)
    adr = ADROracle(o, lam)
    sim = pd.Sim(x, vol, 3.015e-3, **kw, flags=fl, value=val)
    for chunk in (1, 2, 40, 300):
        adr.iterate(chunk); sim.adr_step(chunk, lam)
        assert _rel(sim.get_u(), o.u) <= 1e-9, chunk
    assert np.abs(o.u).max() > 1e-7 and max(adr.c_hist) > 0
    sim.destroy()
    # plate 40 x 24 with a pre-notch; top and bottom rows driven apart by a fixed increment per iteration
    nx, ny, dx = 40, 24, 1e-3
    gx, gy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    gx, gy = gx.reshape(-1), gy.reshape(-1)
    x = np.stack([(gx + 0.5) * dx, (gy + 0.5) * dx], 1)
    fl = np.zeros(nx * ny, np.uint8); val = np.zeros((nx * ny, 2))
    fl[gy >= ny - 3] = 8 | 16; val[gy >= ny - 3, 1] = +2e-9
    fl[gy < 3] = 8 | 16; val[gy < 3, 1] = -2e-9
    from paper_2309_11273_b200.workloads import _precut_horizontal
    precut = _precut_horizontal(nx, ny, ny // 2, 2 * (nx // 3))
    vol = np.full(nx * ny, dx * dx * 1e-3)
    lam = 0.3 * 72e9 / dx ** 2
    # (b) s_c so small that the bonds next to the driven rows break in iterations 4-8 (stretch 2e-6 per iteration)
    kw = dict(dim=2, mode=1, E=72e9, nu=0.22, rho=1.0, dt=1.0, s_c=7e-6)
    o = PDOracle(x, vol, 3.015 * dx, **kw, flags=fl, value=val, precut=precut)
    adr = ADROracle(o, lam)
    sim = pd.Sim(x, vol, 3.015 * dx, **kw, flags=fl, value=val, precut=precut)
    for chunk in (3, 2, 3):
        adr.iterate(chunk); sim.adr_step(chunk, lam)
        bs, _, _ = _broken_set(sim)
        assert adr.near_total == 0, "near-threshold events must be reported"
        assert bs == o.broken_set(), (len(bs), len(o.broken_set()))
        assert _rel(sim.get_u(), o.u) <= 1e-10
        assert np.allclose(sim.get_damage(), o.damage(), rtol=0, atol=1e-12)
    assert len(o.broken_set()) > 2 * len(precut), "the case must actually break bonds"
    sim.destroy()
    # (c) no failure: 100 increments, then hold and relax: both reach the same equilibrium
    kw["s_c"] = 0.0
    o = PDOracle(x, vol, 3.015 * dx, **kw, flags=fl, value=val, precut=precut)
    adr = ADROracle(o, lam)
    sim = pd.Sim(x, vol, 3.015 * dx, **kw, flags=fl, value=val, precut=precut)
    adr.iterate(100); sim.adr_step(100, lam)
    sim.destroy()
    u_hold = o.u.copy()
    o2 = PDOracle(x, vol, 3.015 * dx, **kw, flags=fl, value=np.zeros_like(val), precut=precut, u0=u_hold)
    # (prescribed dofs keep the displacement reached; increments are zero from here on)
    adr2 = ADROracle(o2, lam)
    sim2 = pd.Sim(x, vol, 3.015 * dx, **kw, flags=fl, value=np.zeros_like(val), precut=precut, u0=u_hold)
    adr2.iterate(2500); sim2.adr_step(2500, lam)
    assert _rel(sim2.get_u(), o2.u) <= 1e-6
    r = np.abs(adr2.total_force()[(fl & 24) == 0]).max()       # residual on the free dofs at the oracle's end state
    assert r <= 1e-6 * np.abs(adr2.o.force_density()).max()
    sim2.destroy()
