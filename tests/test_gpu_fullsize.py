"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default
renumbering, persistent kernels with their full resident grids): the whole state after a few time
steps against the oracle run on the host cores, plus the RHS and flux buffer on the full mesh.

The oracle needs about a second per RK stage at these sizes, so the step counts are small; the long
runs are covered on the small meshes of test_gpu_parity.py.
"""
import numpy as np
import pytest

from workloads import c2, c3, c4, c5, perturbed

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-12
STATE_TOL = 1e-10


@pytest.fixture(scope="module")
def G():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_21208_b200 import build
    build.build()
    import paper_2508_21208_b200 as pk
    return pk


def full_size_case(O, G, w, nsteps):
    o = O.Oracle.from_workload(w)
    g = G.Dgswem.from_workload(w, reorder=1)
    assert np.array_equal(g.get_wetdry(), o.get_wetdry())
    r_cpu, s_cpu = o.eval_rhs(with_scale=True)
    r_gpu = g.eval_rhs()
    f_cpu, f_gpu = o.get_flux(), g.get_flux()
    assert np.array_equal(f_gpu, f_cpu)
    for c in range(3):
        err = np.abs(r_gpu[c] - r_cpu[c]).max() / max(s_cpu[c].max(), 1e-300)
        assert err <= RHS_TOL
        assert np.array_equal(r_gpu[c], r_cpu[c])
    del r_cpu, s_cpu, r_gpu, f_cpu, f_gpu
    o.step(nsteps, w.dt); g.step(nsteps, w.dt)
    t_cpu, *sc = o.get_state()
    t_gpu, *sg = g.get_state()
    assert t_cpu == t_gpu
    for c in range(3):
        den = float(np.sqrt((sc[c] ** 2).sum()))
        num = float(np.sqrt(((sg[c] - sc[c]) ** 2).sum()))
        assert num <= STATE_TOL * (den if den > 0 else 1.0)
        assert np.array_equal(sg[c], sc[c])
    wet_cpu, wet_gpu = o.get_wetdry(), g.get_wetdry()
    assert np.array_equal(wet_gpu, wet_cpu)
    for a, b in zip(g.get_nodal(), o.get_nodal()):
        assert np.array_equal(a, b)
    g.close()
    return sg, wet_gpu


def test_c3_full_size(O, G):
    """BASELINE configs[2], the bench workload: 4,494,002 permuted elements, p=1, M2 tide."""
    w = c3()
    assert w.mesh.n_elem == 4_494_002
    sg, _ = full_size_case(O, G, w, 3)
    assert np.abs(sg[0]).max() > 0


def test_c3_full_size_nonzero_state(O, G):
    """The bench workload's mesh, tide and launch configuration on NON-ZERO data: smooth waves plus seeded noise in all
    three modes of zeta, Qx, Qy (0.3 m / 1 m2/s) in every element, so the 4.49 M-element permuted neighbour gather,
    the Hilbert renumbering and every mode are compared on values that differ from element to element (from rest,
    3 steps move only the east boundary column).  RHS, flux buffer, state, mask and nodal output bit for bit."""
    w = perturbed(c3())
    assert w.mesh.n_elem == 4_494_002
    assert min(np.abs(a).min() for a in (w.ze, w.qx, w.qy)) > 0
    sg, _ = full_size_case(O, G, w, 3)
    assert all(np.abs(a).min() > 0 for a in sg)


def test_c5_full_size_nonzero_quadratic_modes(O, G):
    """BASELINE configs[4] with all six modes populated offshore (the recipe starts with zero quadratic modes)."""
    w = perturbed(c5(), amp_z=0.2)
    assert np.abs(w.ze[3:]).max() > 1e-3
    full_size_case(O, G, w, 2)


def test_c4_full_size(O, G):
    """BASELINE configs[3]: 1,048,576 elements, ~20 % dry, wind + limiter + wet/dry."""
    w = c4()
    assert w.mesh.n_elem == 1_048_576
    _, wet = full_size_case(O, G, w, 6)
    assert 0.1 < 1.0 - wet.mean() < 0.3


def test_c5_full_size(O, G):
    """BASELINE configs[4]: ~3.5 M elements, p=2, RK3, everything on."""
    w = c5()
    assert w.mesh.n_elem > 3_400_000
    full_size_case(O, G, w, 1)


@pytest.mark.parametrize("p", [1, 2])
def test_c2_full_size(O, G, p):
    """BASELINE configs[1]: 524,288 elements, p = 1 and 2, friction + Coriolis."""
    w = c2(p=p)
    assert w.mesh.n_elem == 524_288
    full_size_case(O, G, w, 4)


def test_c2_full_size_p3(O, G):
    """The C2 mesh at p = 3, all ten modes populated."""
    w = perturbed(c2(p=3), amp_z=0.2)
    assert w.mesh.n_elem == 524_288 and np.abs(w.ze[6:]).max() > 1e-3
    full_size_case(O, G, w, 2)
