"""Domain decomposition: a run split into partitions with one layer of
ghost elements, stepped through the stage-granular C ABI with a halo exchange per RK stage (and one of the means before
the limiter pass), must reproduce the undivided run BIT FOR BIT on every owned element -- state, time and wet/dry mask.
All partitions live on the one GPU of this box (LocalTransport); the multi-rank transport is covered on CPU in
tests/test_partition.py."""
import numpy as np
import pytest

from workloads import c2, c3, c4, c5, perturbed

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_21208_b200 import build
    build.build()
    import paper_2508_21208_b200 as pk
    return pk


CASES = {
    "c3-nonzero-state": lambda: perturbed(c3(nn=40, nsteps=25)),
    "c3-tide-wetdry": lambda: c3(nn=40, nsteps=25),
    "c4-limiter-wind": lambda: c4(nqx=48, nqy=24, nsteps=40),
    "c5-p2-rk3-all": lambda: c5(nn=30, nsteps=20),
    "c2-p1-friction": lambda: c2(nq=24, p=1, state="hump", nsteps=20),
}


@pytest.mark.parametrize("fused", ["0", "1", "1-no-overlap", "2", "3"],
                         ids=["edge+elem", "stage", "stage-no-overlap", "stage-tile", "stage-staged"])   # overlap is forced on otherwise
@pytest.mark.parametrize("n_parts", [2, 5])
@pytest.mark.parametrize("case", sorted(CASES))
def test_partitioned_run_equals_undivided_run(O, G, monkeypatch, case, n_parts, fused):
    """... and the ORACLE's run, directly (not only transitively through the undivided GPU run).  By default every stage
    is split into the send-list elements (dgswem_stage_rhs_part 1), whose packed values travel on the communication
    stream while the interior elements are computed (part 2); "no-overlap" is the unsplit order of calls."""
    overlap = not fused.endswith("no-overlap")
    fused = fused[0]
    from paper_2508_21208_b200.decomp import PartitionedDgswem
    monkeypatch.setenv("DGSWEM_FUSED", fused)
    w = CASES[case]()
    m = w.mesh
    o = O.Oracle.from_workload(w)
    o.step(w.nsteps, w.dt)
    t_orc, *s_orc = o.get_state()
    wet_orc = o.get_wetdry()
    ref = G.Dgswem.from_workload(w, reorder=1)
    ref.step(w.nsteps, w.dt)
    t_ref, *s_ref = ref.get_state()
    wet_ref = ref.get_wetdry()
    ref.close()
    pd = PartitionedDgswem(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, n_parts,
                           tide=w.tide, holland=w.holland, overlap=overlap)
    assert sum(s.n_owned for s in pd.subs) == m.n_elem
    assert all(s.n_local > s.n_owned for s in pd.subs)            # every partition has ghosts
    pd.set_state(0.0, w.ze, w.qx, w.qy)
    pd.step(w.nsteps, w.dt)
    t, *s = pd.get_state()
    assert t == t_ref
    for c in range(3):
        assert np.array_equal(s[c], s_ref[c])
    assert np.array_equal(pd.get_wetdry(), wet_ref)
    assert t == t_orc and np.array_equal(pd.get_wetdry(), wet_orc)
    for c in range(3):
        assert np.array_equal(s[c], s_orc[c])
    pd.close()


@pytest.mark.parametrize("overlap", [False, True], ids=["unsplit", "overlap"])
@pytest.mark.parametrize("case", ["c3-tide-wetdry", "c4-limiter-wind", "c5-p2-rk3-all"])
def test_partitioned_step_recorded_as_one_cuda_graph(O, G, case, overlap):
    """graph=True: one CUDA graph holds a whole decomposed step (three partitions' kernels, packs, copies, unpacks and
    their dependencies; dgswem_capture_mode), replayed for every step with the tide / storm-centre scalars read from the
    handles' device tables (dgswem_graph_steps), in two calls so that the tables are refilled at a later time.  Same bits
    as the oracle's undivided run."""
    from paper_2508_21208_b200.decomp import PartitionedDgswem
    w = CASES[case]()
    m = w.mesh
    o = O.Oracle.from_workload(w)
    o.step(w.nsteps, w.dt)
    t_orc, *s_orc = o.get_state()
    pd = PartitionedDgswem(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, 3,
                           tide=w.tide, holland=w.holland, overlap=overlap, graph=True)
    pd.set_state(0.0, w.ze, w.qx, w.qy)
    l0 = sum(g.launch_count() for g in pd.handles)
    first = w.nsteps // 3
    pd.step(first, w.dt)
    pd.step(w.nsteps - first, w.dt)
    t, *s = pd.get_state()
    assert t == t_orc
    for c in range(3):
        assert np.array_equal(s[c], s_orc[c])
    assert np.array_equal(pd.get_wetdry(), o.get_wetdry())
    assert pd._graph is not None
    pd.close()


def test_stage_api_equals_dgswem_step_and_rejects_misuse(G):
    """begin_step / stage_rhs / stage_limit / end_step on an undivided mesh (no halo) is dgswem_step; misuse is an error."""
    w = c4(nqx=32, nqy=16, nsteps=15)
    a = G.Dgswem.from_workload(w)
    b = G.Dgswem.from_workload(w)
    a.step(15, w.dt)
    for _ in range(15):
        b.begin_step(w.dt)
        for s in range(w.n_stage):
            b.stage_rhs(s); b.stage_limit(s)
        b.end_step()
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(x, y)
    with pytest.raises(G.DgswemError):
        b.stage_rhs(0)                      # no step in progress
    b.begin_step(w.dt)
    with pytest.raises(G.DgswemError):
        b.step(1, w.dt)                     # dgswem_step inside a stage-granular step
    with pytest.raises(G.DgswemError):
        b.stage_rhs(7)
    with pytest.raises(G.DgswemError):
        b.stage_rhs(0, part=3)
    with pytest.raises(G.DgswemError):
        b.capture_mode(True)                # not inside a step
    b.end_step()
    b.capture_mode(True)
    with pytest.raises(G.DgswemError):
        b.step(1, w.dt)                     # dgswem_step while the handle records for the caller's graph
    with pytest.raises(G.DgswemError):
        b.graph_steps(1, w.dt)
    b.capture_mode(False)
    with pytest.raises(G.DgswemError):
        b.graph_steps(5000, w.dt)           # more rows than the scalar table holds
    a.close(); b.close()


def test_capture_mode_refuses_calls_that_synchronise(G):
    """While a stage-granular step is being recorded into the caller's graph (dgswem_capture_mode(1)) a call that
    synchronises the handle's stream would invalidate the capture: such calls are refused with DGSWEM_E_ARG and work
    again once capture mode is off."""
    w = c3(nn=20, nsteps=2)
    g = G.Dgswem.from_workload(w)
    g.capture_mode(True)
    for call in (g.get_state, g.get_wetdry, g.get_nodal, g.eval_rhs, g.get_flux, g.sync, lambda: g.step(1, w.dt),
                 lambda: g.set_state(0.0, w.ze, w.qx, w.qy)):
        with pytest.raises(G.DgswemError, match="capture mode") as ei:
            call()
        assert ei.value.code == -1
    g.capture_mode(False)
    g.step(2, w.dt)
    t, *_ = g.get_state()
    assert t == 2 * w.dt
    g.close()


def _with_params(w, **kw):
    from workloads.configs import Workload
    prm = dict(w.params); prm.update(kw)
    return Workload(w.name, w.mesh, w.bathy, prm, w.ze, w.qx, w.qy, w.dt, w.nsteps, tide=w.tide, holland=w.holland, notes=w.notes)


VARIANTS = {
    "roe": lambda: _with_params(c4(nqx=48, nqy=24, nsteps=30), flux=1),
    "ssp43": lambda: _with_params(c5(nn=30, nsteps=16), rk_stages=4),
    "ssp42-p1": lambda: _with_params(perturbed(c3(nn=40, nsteps=20)), rk_stages=4),
    "p3": lambda: perturbed(c5(nn=30, nsteps=12, p=3), amp_z=0.2),
    "pressure-rain": lambda: __import__("workloads").with_forcing(c5(nn=30, nsteps=16, p=1, rk_order=2), pressure=True, rain=2.5e-5),
    "f32": lambda: c4(nqx=48, nqy=24, nsteps=30),
    # vertex-neighbourhood limiter: partitions with a vertex ghost layer (every foreign element around an owned node)
    "vertexlim-c4": lambda: _with_params(perturbed(c4(nqx=48, nqy=24, nsteps=30), amp_z=0.2), limiter=2),
    "vertexlim-c5p2": lambda: _with_params(perturbed(c5(nn=30, nsteps=16), amp_z=0.2), limiter=2),
}


@pytest.mark.parametrize("graph", [False, True], ids=["stream", "graph"])
@pytest.mark.parametrize("variant", sorted(VARIANTS))
def test_partitioned_run_of_the_method_variants(O, G, variant, graph):
    """Roe flux, many-stage SSP-RK, p = 3, pressure-gradient + rain forcing and binary32 working precision in a
    decomposed run (three partitions, PartitionedDgswem.from_workload, which hands every forcing of the workload to
    every handle): owned elements bit-equal to the oracle's undivided run (the binary32 oracle for precision 32)."""
    from paper_2508_21208_b200.decomp import PartitionedDgswem
    w = VARIANTS[variant]()
    if variant == "f32":
        from oracle import oracle32
        oracle32.build()
        o = oracle32.Oracle.from_workload(w)
    else:
        o = O.Oracle.from_workload(w)
    o.step(w.nsteps, w.dt)
    t_orc, *s_orc = o.get_state()
    pd = PartitionedDgswem.from_workload(w, 3, graph=graph, precision=32 if variant == "f32" else 64)
    pd.step(w.nsteps, w.dt)
    t, *s = pd.get_state()
    assert t == t_orc
    for c in range(3):
        assert np.isfinite(s_orc[c]).all() and np.array_equal(s[c], np.asarray(s_orc[c], dtype=np.float64))
    assert np.array_equal(pd.get_wetdry(), o.get_wetdry())
    pd.close()
