"""Pins for the binary32 build of the oracle (oracle/oracle32.py, PAPER.md:158 "-r4", :529 "computation
is done with single-precision").  It is the same source as the pinned binary64 oracle with `real` = float, so it is pinned
(a) against closed forms at binary32 tolerances and (b) against the binary64 oracle, which the rest of tests/ pins."""
import math

import numpy as np
import pytest

from helpers import G, phys_flux, small_mesh
from workloads import c2, c3, c4, c5, default_params, perturbed

EPS = float(np.finfo(np.float32).eps)      # 1.19e-7


@pytest.fixture(scope="module")
def O32():
    from oracle import oracle32
    oracle32.build()
    return oracle32


def test_f32_tables_closed_forms(O32):
    """Mass M_ij = 2/((2i+1)(i+j+1)) folded into the weights, vertex values of the basis, weights summing to 2."""
    for p in (1, 2):
        T = O32.tables(p)
        nd = (p + 1) * (p + 2) // 2
        M = np.array([2.0, 1.0, 1 / 3, 2 / 3, 2 / 9, 2 / 15])[:nd]
        assert np.abs(T.np("invM")[:nd] - 1 / M).max() <= 2 * EPS * 8
        assert abs(T.np("wa")[:T.nqa].sum() - 2.0) <= 4 * EPS and abs(T.np("we")[:T.nqe].sum() - 2.0) <= 4 * EPS
        V = np.array([[1, 1, 1], [-1, -1, 2], [-1, 1, 0], [1, 1, 3], [1, -1, 0], [1, 1, 0]], dtype=float)[:nd]
        assert np.abs(T.np("phiV")[:, :nd].T - V).max() <= 8 * EPS
        # discrete orthogonality of the area rule (exact to degree 2p): sum_i wa_i phi_k phi_l = M_k delta_kl
        phiA, wa = T.np("phiA")[:T.nqa, :nd].astype(float), T.np("wa")[:T.nqa].astype(float)
        assert np.abs((phiA * wa[:, None]).T @ phiA - np.diag(M)).max() <= 32 * EPS
        assert T.np("phiA").dtype == np.float32


def test_f32_flux_consistency_and_antisymmetry(O32):
    rng = np.random.default_rng(0)
    for _ in range(100):
        th = rng.uniform(0, 2 * np.pi); n = (np.float32(math.cos(th)), np.float32(math.sin(th)))
        h = rng.uniform(1, 50)
        w = [rng.uniform(-1, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        w2 = [rng.uniform(-1, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        Fx, Fy = phys_flux(*[np.float64(x) for x in w], h, 1e-3)
        ex = Fx * float(n[0]) + Fy * float(n[1])
        for fl in (O32.llf_flux, O32.roe_flux):
            f = fl(G, 1e-3, n[0], n[1], h, w, w)
            assert np.abs(f - ex).max() <= 64 * EPS * max(1.0, np.abs(ex).max())          # F^(w, w) = F(w).n
            f1 = fl(G, 1e-3, n[0], n[1], h, w, w2)
            f2 = fl(G, 1e-3, -n[0], -n[1], h, w2, w)
            assert np.array_equal(f1, -f2)                                                # bitwise, as in binary64
            assert fl(G, 1e-3, n[0], n[1], h, w, [9, 9, 9], bc=1)[0] == 0.0               # wall mass flux exactly 0


def test_f32_det_exp_log(O32):
    rng = np.random.default_rng(1)
    for x in rng.uniform(-30, 30, 300):
        assert abs(O32.det_exp(x) - math.exp(np.float32(x))) <= 64 * EPS * math.exp(np.float32(x))
    for x in 10 ** rng.uniform(-6, 6, 300):
        assert abs(O32.det_log(x) - math.log(np.float32(x))) <= 16 * EPS * max(1.0, abs(math.log(x)))
    assert O32.det_exp(-100.0) == 0.0


@pytest.mark.parametrize("p", [1, 2])
def test_f32_lake_at_rest_and_mass(O32, p):
    w = c2(nq=12, p=p, state="rest")
    o = O32.Oracle.from_workload(w)
    r, s = o.eval_rhs(with_scale=True)
    for c in range(3):
        assert np.abs(r[c]).max() <= 64 * EPS * max(float(s[c].max()), 1.0)
    w = c2(nq=12, p=p, state="hump")
    o = O32.Oracle.from_workload(w)
    area = o.get_geometry()[0].astype(float)
    m0 = float((area * w.ze[0]).sum())
    o.step(40, w.dt)
    _, ze, qx, qy = o.get_state()
    assert ze.dtype == np.float32 and np.isfinite(ze).all() and np.abs(qx).max() > 1e-3
    # closed walls: the mass error is rounding only (the mean depth ~10-50 m carries eps = 1.2e-7 per update)
    assert abs(float((area * ze[0].astype(float)).sum()) - m0) < 1e-5 * area.sum() * 0.5


@pytest.mark.parametrize("recipe", ["c2p1", "c2p2", "c3", "c4", "c5"])
def test_f32_tracks_the_binary64_oracle(O, O32, recipe):
    """Same inputs, same steps: relative L2 distance of the binary32 run from the pinned binary64 run stays at the
    level of accumulated binary32 rounding (<= 2e-5 after these step counts; a formula difference would be O(1e-2+)),
    and the wet/dry masks agree except where a depth sits within rounding of a threshold."""
    w = {"c2p1": lambda: perturbed(c2(nq=24, p=1, state="hump", nsteps=40), amp_z=0.2),
         "c2p2": lambda: perturbed(c2(nq=24, p=2, state="hump", nsteps=40), amp_z=0.2),
         "c3": lambda: perturbed(c3(nn=40, nsteps=40)), "c4": lambda: c4(nqx=48, nqy=24, nsteps=60),
         "c5": lambda: c5(nn=30, nsteps=30)}[recipe]()
    o, o32 = O.Oracle.from_workload(w), O32.Oracle.from_workload(w)
    assert (o.get_wetdry() != o32.get_wetdry()).mean() <= 0.01
    o.step(w.nsteps, w.dt); o32.step(w.nsteps, w.dt)
    t, *s = o.get_state(); t32, *s32 = o32.get_state()
    assert t == t32                                           # time is binary64 in both builds
    for a, b in zip(s, s32):
        den = math.sqrt(float((a * a).sum()))
        assert math.sqrt(float(((a - b.astype(float)) ** 2).sum())) <= 2e-5 * max(den, 1.0)
    assert (o.get_wetdry() != o32.get_wetdry()).mean() <= 0.01
    for a, b in zip(o.get_nodal(), o32.get_nodal()):
        assert np.abs(a - b).max() <= 1e-4 * max(1.0, np.abs(a).max())
