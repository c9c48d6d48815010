"""The L2-prefetching variants of the element-centric stage kernel (k_stage<..., PF = 1>, csrc/dgswem_impl.inl
launch_stage) against the oracle.  By default the prefetch switches on only for meshes whose stage buffer exceeds
100 MB, so of all its instantiations -- (first stage?) x (wind, pressure, rain, generic flags), each in binary64 and in
binary32 -- only the no-wind binary64 pair is reached by the full-size C3 cases.  DGSWEM_PF_DIST forces a distance on the
small recipes here (1-3 tiles of 128 elements, so that the "is there a tile that far ahead" guard is crossed at the
ragged end of every mesh), one recipe per specialisation, in both precisions.  Prefetches are hints: the bits must not
change (the fp32 headline rows of BASELINE.md run exactly these kernels)."""
import numpy as np
import pytest

from workloads import c2, c3, c4, c5, perturbed, with_forcing
from workloads.configs import Workload

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


@pytest.fixture(scope="module")
def O32():
    from oracle import oracle32
    oracle32.build()
    return oracle32


def _with_params(w, **kw):
    prm = dict(w.params); prm.update(kw)
    return Workload(w.name, w.mesh, w.bathy, prm, w.ze, w.qx, w.qy, w.dt, w.nsteps, tide=w.tide, holland=w.holland, notes=w.notes)


# one recipe per specialisation of the p = 1 stage kernel: plain, friction + Coriolis, tide + wet/dry, wind + limiter,
# wind + pressure + rain, RK3, SSP(4,3) (plain stages without a w^n read in the middle of the step)
RECIPES = {
    "c2p1-hump": lambda: perturbed(c2(nq=41, p=1, state="hump", nsteps=20), amp_z=0.2),
    "c3": lambda: perturbed(c3(nn=60, nsteps=20)),
    "c4": lambda: c4(nqx=64, nqy=32, nsteps=40),
    "c4-perturbed": lambda: perturbed(c4(nqx=64, nqy=32, nsteps=20), amp_z=0.2),
    "c5p1-pressure-rain": lambda: with_forcing(c5(nn=40, nsteps=20, p=1, rk_order=2), pressure=True, rain=2.5e-5),
    "c5p1-rk3": lambda: c5(nn=40, nsteps=20, p=1, rk_order=3),
    "c5p1-ssp43": lambda: _with_params(c5(nn=40, nsteps=20, p=1, rk_order=3), rk_stages=4),
}


@pytest.mark.parametrize("pf_dist", ["1", "3"])
@pytest.mark.parametrize("graph", ["1", "0"])
@pytest.mark.parametrize("recipe", sorted(RECIPES))
def test_prefetching_stage_kernels_fp64(O, G, monkeypatch, recipe, graph, pf_dist):
    monkeypatch.setenv("DGSWEM_FUSED", "1")
    monkeypatch.setenv("DGSWEM_PF_DIST", pf_dist)
    monkeypatch.setenv("DGSWEM_GRAPH", graph)
    w = RECIPES[recipe]()
    assert w.mesh.n_elem % 128 != 0 or recipe.startswith("c4")     # ragged last tile (the C4 channel is 4096 elements)
    o = O.Oracle.from_workload(w)
    g = G.Dgswem.from_workload(w, reorder=1)
    assert g.stage_form() == 1
    for a, b in zip(g.eval_rhs(), o.eval_rhs()):
        assert np.array_equal(a, b)
    half = w.nsteps // 2
    for n in (half, w.nsteps - half):
        o.step(n, w.dt); g.step(n, w.dt)
    t_cpu, *s_cpu = o.get_state()
    t_gpu, *s_gpu = g.get_state()
    assert t_cpu == t_gpu
    for c in range(3):
        assert np.isfinite(s_cpu[c]).all() and np.array_equal(s_gpu[c], s_cpu[c])
    assert np.array_equal(g.get_wetdry(), o.get_wetdry())
    g.close()


@pytest.mark.parametrize("recipe", ["c3", "c4-perturbed", "c5p1-pressure-rain"])
def test_prefetching_stage_kernels_fp32(O32, G, monkeypatch, recipe):
    monkeypatch.setenv("DGSWEM_FUSED", "1")
    monkeypatch.setenv("DGSWEM_PF_DIST", "2")
    w = RECIPES[recipe]()
    o = O32.Oracle.from_workload(w)
    g = G.Dgswem.from_workload(w, reorder=1, precision=32)
    assert g.stage_form() == 1 and g.precision() == 32
    wide = lambda a: np.asarray(a, dtype=np.float64)
    o.step(w.nsteps, w.dt); g.step(w.nsteps, w.dt)
    _, *s_cpu = o.get_state()
    _, *s_gpu = g.get_state()
    for c in range(3):
        assert np.isfinite(s_cpu[c]).all() and np.array_equal(s_gpu[c], wide(s_cpu[c]))
    assert np.array_equal(g.get_wetdry(), o.get_wetdry())
    g.close()


def test_c3_full_size_fp32(O32, G):
    """BASELINE configs[2] at full size in binary32 -- the C3_f32 row of BASELINE.md, in the launch configuration
    bench.py --dtype f32 times (prefetching k_stage, graph replay) -- against the binary32 oracle: 3 steps from a
    non-zero state, state and mask bit for bit."""
    w = perturbed(c3())
    assert w.mesh.n_elem == 4_494_002
    o = O32.Oracle.from_workload(w)
    g = G.Dgswem.from_workload(w, reorder=1, precision=32)
    o.step(3, w.dt); g.step(3, w.dt)
    _, *s_cpu = o.get_state()
    _, *s_gpu = g.get_state()
    for c in range(3):
        assert np.isfinite(s_cpu[c]).all()
        assert np.array_equal(s_gpu[c], np.asarray(s_cpu[c], dtype=np.float64))
    assert np.array_equal(g.get_wetdry(), o.get_wetdry())
    g.close()
