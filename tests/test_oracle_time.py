"""Pins for the oracle's time stepping, conservation, limiter, wet/dry and wind.
PAPER.md:109 (SSP-RK, limiter), :326 (SLOPELIM, WETDRY, WIND); SURVEY.md §8(c.5)."""
import math

import numpy as np
import pytest

from helpers import G, l2_project, small_mesh
from workloads import c1, c2, c4, default_params
from workloads.mesh import rect_mesh
from workloads.mesh import vertex_to_modal_p1


# ------------------------------------------------------------------ SSP-RK
@pytest.mark.parametrize("order", [2, 3])
def test_ssprk_order_on_linear_decay(O, order):
    """dw/dt = -w, w(0)=1 to t=1: halving dt divides the error by 2^order."""
    errs = []
    for n in (20, 40, 80):
        w = np.array([1.0, -2.0])
        dt = 1.0 / n
        for i in range(n):
            w = O.ssprk_step(order, w, i * dt, dt, lambda s, ts, ww: -ww)
        errs.append(abs(w[0] - math.exp(-1.0)))
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert abs(math.log2(r1) - order) < 0.15 and abs(math.log2(r2) - order) < 0.1


def test_ssprk_stage_times_and_exact_stage_polynomials(O):
    """Stage times c = (0,1) / (0,1,1/2); for dw/dt = lambda w one step multiplies by the
    degree-`order` Taylor polynomial of exp(lambda dt)."""
    for order, cs in ((2, [0.0, 1.0]), (3, [0.0, 1.0, 0.5])):
        seen = []
        O.ssprk_step(order, np.array([1.0]), 10.0, 0.5, lambda s, ts, ww: (seen.append(ts), 0.0 * ww)[1])
        assert np.allclose(seen, [10.0 + c * 0.5 for c in cs], atol=0)
        z = -0.3
        w = O.ssprk_step(order, np.array([1.0]), 0.0, 1.0, lambda s, ts, ww: z * ww)
        taylor = sum(z ** k / math.factorial(k) for k in range(order + 1))
        assert abs(w[0] - taylor) < 1e-15


# many-stage schemes (reading R-19): (order, stages) and the textbook stability polynomial of each, i.e. the factor one
# step applies to dw/dt = lambda w: SSP(s,2): 1/s + (s-1)/s (1 + z/(s-1))^s; SSP(4,3): 2/3 (1 + z/2) + 1/3 (1 + z/2)^4,
# written out in powers of z
MANY_STAGE = {(2, 3): ([0.0, 0.5, 1.0], [1.0, 1.0, 0.5, 1.0 / 12.0]),
              (2, 4): ([0.0, 1.0 / 3.0, 2.0 / 3.0, 1.0], [1.0, 1.0, 0.5, 1.0 / 9.0, 1.0 / 108.0]),
              (3, 4): ([0.0, 0.5, 1.0, 0.5], [1.0, 1.0, 0.5, 1.0 / 6.0, 1.0 / 48.0])}


@pytest.mark.parametrize("scheme", sorted(MANY_STAGE))
def test_many_stage_ssprk_stability_polynomial_and_stage_times(O, scheme):
    order, stages = scheme
    cs, poly = MANY_STAGE[scheme]
    seen = []
    O.ssprk_step(order, np.array([1.0]), 10.0, 0.5, lambda s, ts, ww: (seen.append(ts), 0.0 * ww)[1], stages=stages)
    assert len(seen) == stages and np.allclose(seen, [10.0 + c * 0.5 for c in cs], rtol=0, atol=1e-15)
    for z in (-0.3, 0.7, -1.9):
        w = O.ssprk_step(order, np.array([1.0, -2.0]), 0.0, 1.0, lambda s, ts, ww: z * ww, stages=stages)
        exact = sum(ck * z ** k for k, ck in enumerate(poly))
        assert abs(w[0] - exact) < 4e-16 * max(1.0, abs(exact)) * 8 and abs(w[1] + 2.0 * exact) < 1e-14
    # the polynomial matches exp(z) through z^order and not beyond
    for k in range(order + 1):
        assert abs(poly[k] - 1.0 / math.factorial(k)) < 1e-15
    assert abs(poly[order + 1] - 1.0 / math.factorial(order + 1)) > 1e-3


@pytest.mark.parametrize("scheme", sorted(MANY_STAGE))
def test_many_stage_ssprk_order_with_time_dependent_forcing(O, scheme):
    """dw/dt = -w + cos t, w(0) = 0, exact w = (cos t + sin t - exp(-t)) / 2: the observed order is the scheme's,
    which needs both the stage weights and the stage times to be right."""
    order, stages = scheme
    errs = []
    for n in (16, 32, 64):
        w = np.array([0.0]); dt = 2.0 / n
        for i in range(n):
            w = O.ssprk_step(order, w, i * dt, dt, lambda s, ts, ww: -ww + math.cos(ts), stages=stages)
        errs.append(abs(w[0] - 0.5 * (math.cos(2.0) + math.sin(2.0) - math.exp(-2.0))))
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert abs(math.log2(r1) - order) < 0.25 and abs(math.log2(r2) - order) < 0.15, (errs, r1, r2)


def test_many_stage_ssprk_is_ssp_with_larger_step(O):
    """Strong stability: with L the first-order upwind operator on a periodic grid (forward Euler is TVD for
    nu = a dt / dx <= 1), SSP(s,2) stays TVD up to nu = s - 1 and SSP(4,3) up to nu = 2 (the schemes' SSP coefficients,
    which is what "optimized" buys), and each loses it a little beyond: a square wave's total variation is the witness."""
    n = 64
    u0 = np.where((np.arange(n) >= 16) & (np.arange(n) < 40), 1.0, 0.0)
    tv = lambda u: np.abs(u - np.roll(u, 1)).sum()
    up = lambda s, ts, u: -(u - np.roll(u, 1))          # a / dx = 1: dt is the Courant number
    for (order, stages), c_ssp in (((2, 2), 1.0), ((3, 3), 1.0), ((2, 3), 2.0), ((2, 4), 3.0), ((3, 4), 2.0)):
        for nu, must_hold in ((c_ssp, True), (1.6 * c_ssp, False)):
            u = u0.copy(); worst = 0.0
            for i in range(40):
                u = O.ssprk_step(order, u, 0.0, nu, up, stages=stages)
                worst = max(worst, tv(u) - tv(u0))
            assert (worst <= 1e-12) == must_hold, (order, stages, nu, worst)


def test_many_stage_scheme_in_the_model(O):
    """The model takes rk_stages: seiche amplitude after a fixed time agrees between SSP(3,3) at dt and SSP(4,3) at
    2 dt to the schemes' third-order accuracy, and an unknown (order, stages) pair is refused."""
    mesh = rect_mesh(8, 8, 1000.0, 1000.0)
    H = 10.0
    ze0 = vertex_to_modal_p1(0.01 * np.cos(np.pi * mesh.xy[:, 0] / 1000.0), mesh.tri, 3)
    z = np.zeros_like(ze0)
    res = {}
    for stages, dt, n in ((0, 1.0, 40), (4, 2.0, 20)):
        prm = default_params(p=1, rk_order=3); prm["rk_stages"] = stages
        o = O.Oracle(prm, mesh.xy, np.full(mesh.n_nodes, H), mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)
        o.set_state(0.0, ze0, z, z)
        o.step(n, dt)
        t, ze, _, _ = o.get_state()
        assert t == 40.0
        res[stages] = ze
    assert 1e-9 < np.abs(res[0] - res[4]).max() < 2e-6       # different schemes, same solution to O(dt^3)
    prm = default_params(p=1, rk_order=3); prm["rk_stages"] = 5
    with pytest.raises(Exception):
        O.Oracle(prm, mesh.xy, np.full(mesh.n_nodes, H), mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)


def test_rk_time_dependent_forcing_uses_stage_time(O):
    """dw/dt = cos(t): RK3 integrates it with 3rd-order accuracy only if t_stage is right."""
    errs = []
    for n in (10, 20):
        w = np.array([0.0]); dt = 1.0 / n
        for i in range(n):
            w = O.ssprk_step(3, w, i * dt, dt, lambda s, ts, ww: np.array([math.cos(ts)]))
        errs.append(abs(w[0] - math.sin(1.0)))
    assert 6.0 < errs[0] / errs[1] < 20.0      # >= 3rd order (this quadrature is Simpson-like)


# ------------------------------------------------------------------ seiche (textbook special case)
def _seiche(O, nq, p, amp=1e-4, t_end=300.0):
    L, H = 10_000.0, 10.0
    mesh = rect_mesh(nq, nq, L, L, diag="same")
    k = math.pi / L
    om = k * math.sqrt(G * H)
    o = O.Oracle(default_params(p=p, rk_order=3), mesh.xy, np.full(mesh.n_nodes, H), mesh.tri,
                 mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)
    ze0 = l2_project(O, mesh, lambda x, y: amp * np.cos(k * x), p)
    o.set_state(0.0, ze0, 0 * ze0, 0 * ze0)
    h = L / nq
    dt = 0.1 * h / ((2 * p + 1) * math.sqrt(G * H))
    n = int(math.ceil(t_end / dt)); dt = t_end / n
    o.step(n, dt)
    t, ze, qx, qy = o.get_state()
    zex = l2_project(O, mesh, lambda x, y: amp * np.cos(k * x) * math.cos(om * t), p)
    qex = l2_project(O, mesh, lambda x, y: amp * math.sqrt(G * H) * np.sin(k * x) * math.sin(om * t), p)
    Mref = np.array([2.0, 1.0, 1 / 3, 2 / 3, 2 / 9, 2 / 15, 1 / 2, 1 / 6, 1 / 10, 1 / 14])[:ze.shape[0], None]
    l2 = lambda a: math.sqrt(float((a * a * Mref).sum()))
    return l2(ze - zex) / l2(zex), l2(qx - qex) / l2(qex), om


@pytest.mark.parametrize("p", [1, 2, 3])
def test_seiche_convergence_order(O, p):
    """Small-amplitude standing wave in the closed flat 10 km basin (linear theory: period
    2L/sqrt(gH) = 2019 s): the L2 error of zeta and Qx converges with order ~ p+1."""
    nqs = (8, 16, 32) if p == 1 else (4, 8, 16) if p == 2 else (3, 6, 12)
    ez, eq = [], []
    for nq in nqs:
        # (p = 3 reaches the linear theory's own error, O(amp / H) relative, on these meshes: a smaller wave)
        a, b, om = _seiche(O, nq, p, amp=1e-4 if p < 3 else 1e-7)
        ez.append(a); eq.append(b)
    assert abs(2 * math.pi / om - 2019.0) < 1.0
    for e in (ez, eq):
        o1, o2 = math.log2(e[0] / e[1]), math.log2(e[1] / e[2])
        assert o2 > p + 0.6 and o1 > p + 0.3, (p, e)
    assert ez[-1] < (2e-3 if p == 1 else 2e-4 if p == 2 else 1e-5)


def test_seiche_period(O):
    """Quarter period: the first-mode amplitude crosses zero at T/4 = 504.8 s."""
    L, H, amp = 10_000.0, 10.0, 1e-4
    mesh = rect_mesh(16, 16, L, L, diag="same")
    o = O.Oracle(default_params(p=2, rk_order=3), mesh.xy, np.full(mesh.n_nodes, H), mesh.tri,
                 mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)
    k = math.pi / L
    ze0 = l2_project(O, mesh, lambda x, y: amp * np.cos(k * x), 2)
    o.set_state(0.0, ze0, 0 * ze0, 0 * ze0)
    area = o.get_geometry()[0]
    cx = mesh.xy[mesh.tri].mean(axis=1)[:, 0]
    shape = np.cos(k * cx)
    dt, prev, tprev, tcross = 2.0, None, None, None
    for i in range(300):
        o.step(1, dt)
        t, ze, _, _ = o.get_state()
        a = float((area * shape * ze[0]).sum())
        if prev is not None and prev > 0 >= a:
            tcross = tprev + (t - tprev) * prev / (prev - a)
            break
        prev, tprev = a, t
    assert tcross is not None and abs(tcross - 2019.0 / 4) < 2.5


# ------------------------------------------------------------------ conservation
def test_mass_conservation_closed_walls_with_limiter_and_wetdry(O):
    """Closed walls: sum_e A_e zeta_00,e is constant to round-off, with friction, wind,
    limiter and wet/dry all active (C4 recipe, small)."""
    w = c4(nqx=32, nqy=16, nsteps=60)
    o = O.Oracle.from_workload(w)
    area = o.get_geometry()[0]
    hbar = w.bathy[w.mesh.tri].mean(axis=1)
    _, ze, _, _ = o.get_state()
    m0 = float((area * ze[0]).sum())
    vol = float((area * np.maximum(ze[0] + hbar, 0)).sum())
    wet0 = o.get_wetdry()
    assert 0.1 < 1.0 - wet0.mean() < 0.35          # ~20 % start dry
    o.step(w.nsteps, w.dt)
    _, ze, qx, qy = o.get_state()
    assert np.isfinite(ze).all() and np.isfinite(qx).all()
    assert np.abs(qx).max() > 1e-6                 # the wind moved the water
    assert abs(float((area * ze[0]).sum()) - m0) < 1e-12 * vol


def test_runup_floods_dry_cells_and_conserves_mass(O):
    """A 1 m hump released 800 m off the shoreline of the C4 beach (small recipe, no wind) runs up the slope: dry
    elements become wet (the mask moves -- 60 steps of wind alone do not move it on this small mesh), nothing dries
    that was wet under still water, and the total mass is conserved to round-off through limiter and wet/dry."""
    from workloads.configs import _modal
    w = c4(nqx=32, nqy=16)
    m = w.mesh
    x = m.xy[:, 0]
    xs = 0.8 * x.max()                                   # h_b = 0 there
    zn = np.maximum(0.5e-3 - w.bathy, 1.0 * np.exp(-((x - (xs - 800.0)) / 400.0) ** 2))
    ze = _modal(zn, m, 1)
    o = O.Oracle(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    o.set_state(0.0, ze, 0 * ze, 0 * ze)
    area = o.get_geometry()[0]
    wet0 = o.get_wetdry()
    _, z0, _, _ = o.get_state()
    m0 = float((area * z0[0]).sum())
    vol = float((area * np.maximum(z0[0] + w.bathy[m.tri].mean(axis=1), 0)).sum())
    o.step(150, w.dt)
    _, z, qx, qy = o.get_state()
    wet1 = o.get_wetdry()
    assert np.isfinite(z).all() and np.isfinite(qx).all() and np.isfinite(qy).all()
    assert (wet1 > wet0).sum() >= 15 and (wet1 < wet0).sum() == 0
    # the newly wet elements lie landward of the initial shoreline
    assert m.xy[m.tri[wet1 > wet0]][:, :, 0].mean(axis=1).min() > xs - 200.0
    assert abs(float((area * z[0]).sum()) - m0) < 1e-13 * vol


def test_hump_mass_and_symmetry_c1(O):
    w = c1(nq=16, nsteps=50)
    o = O.Oracle.from_workload(w)
    area = o.get_geometry()[0]
    _, ze, _, _ = o.get_state()
    m0 = float((area * ze[0]).sum())
    o.step(w.nsteps, w.dt)
    _, ze, qx, qy = o.get_state()
    assert abs(float((area * ze[0]).sum()) - m0) < 1e-13 * 1e9
    assert ze[0].max() < 0.5 and np.abs(qx).max() > 0.1


# ------------------------------------------------------------------ limiter
def test_limiter_properties(O):
    rng = np.random.default_rng(0)
    phiV = np.array([[1, -1, -1], [1, -1, 1], [1, 2, 0]], dtype=float)
    n_active = 0
    for _ in range(300):
        w = rng.normal(size=3) * [1.0, 0.5, 0.5]
        mn = w[0] + rng.normal(size=3) * 0.4
        has = rng.integers(0, 2, 3)
        alpha, wl = O.limit_var(1, w, mn, has)
        assert 0.0 <= alpha <= 1.0
        assert wl[0] == w[0]                                    # mean untouched
        nb = [mn[l] for l in range(3) if has[l]]
        umin, umax = min([w[0]] + nb), max([w[0]] + nb)
        v = phiV @ wl
        assert (v <= umax + 1e-14).all() and (v >= umin - 1e-14).all()
        v0 = phiV @ w
        if (v0 <= umax).all() and (v0 >= umin).all():
            assert alpha == 1.0 and np.array_equal(wl, w)      # no-op when already inside
        else:
            n_active += 1
            assert alpha < 1.0
        a2, wl2 = O.limit_var(1, wl, mn, has)                  # idempotent
        assert np.allclose(wl2, wl, rtol=0, atol=1e-15)
    assert n_active > 50
    # p=2: quadratic modes zeroed iff alpha < 1
    a, wl = O.limit_var(2, [1.0, 2.0, 0.0, 0.3, 0.2, 0.1], [1.1, 0.9, 1.0], [1, 1, 1])
    assert a < 1 and np.array_equal(wl[3:], [0, 0, 0])
    a, wl = O.limit_var(2, [1.0, 1e-3, 0.0, 0.3, 0.2, 0.1], [1.1, 0.9, 1.0], [1, 1, 1])
    assert a == 1 and np.array_equal(wl[3:], [0.3, 0.2, 0.1])


# (limiter_all through the model: tests/test_oracle_pins_sources_post.py)


# ------------------------------------------------------------------ wet/dry
def _vertex(w3):
    return np.array([w3[0] - w3[1] - w3[2], w3[0] - w3[1] + w3[2], w3[0] + 2 * w3[1]])


def test_wetdry_cases(O):
    """[R-8] properties: mass always conserved; exact no-op when every vertex is deeper than
    H1 = 10 H0; dry element -> flat film, no momentum; otherwise all vertex depths >= H0, no
    momentum at vertices with depth <= H0, element momentum conserved, thin vertices attenuated;
    depth part idempotent."""
    h0 = 1e-3
    rng = np.random.default_rng(1)
    seen = {"deep": 0, "thin": 0, 3: 0, 4: 0}
    for it in range(3000):
        hv = rng.uniform(-0.5, 0.5, 3)
        scale = 0.02 if it % 3 == 0 else 1.0          # every third sample sits near the threshold
        ze = np.array([rng.uniform(-0.3, 0.6), rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2)])
        if it % 3 == 0:
            Hwant = rng.uniform(-0.002, 0.02, 3)
            u = Hwant - hv; a = u.sum() / 3
            ze = np.array([a, 0.5 * (u[2] - a), 0.5 * (u[1] - u[0])])
        qx = rng.normal(size=3) * scale; qy = rng.normal(size=3) * scale
        H = _vertex(ze) + hv
        wet, z2, x2, y2 = O.wetdry_elem(1, h0, hv, ze, qx, qy)
        H2 = _vertex(z2) + hv
        assert abs(z2[0] - ze[0]) < 1e-15                     # mean depth (mass) conserved
        if (H > h0).all():
            assert wet == 1 and np.array_equal(z2, ze)          # depths untouched
            if (H >= 10 * h0).all():
                seen["deep"] += 1
                assert np.array_equal(x2, qx) and np.array_equal(y2, qy)
                continue
            seen["thin"] += 1
        elif H.mean() <= h0:
            seen[3] += 1
            assert wet == 0 and not x2.any() and not y2.any()
            assert np.allclose(H2, H.mean(), atol=1e-15)       # flat film
            continue
        else:
            seen[4] += 1
            assert wet == 1 and (H2 >= h0 - 1e-15).all()
            w3, z3, _, _ = O.wetdry_elem(1, h0, hv, z2, x2, y2)
            assert w3 == 1 and np.allclose(z3, z2, atol=1e-14)
        wv = np.clip((H2 - h0) / (9 * h0), 0.0, 1.0)
        wv[H2 <= h0] = 0.0
        for q, q2 in ((qx, x2), (qy, y2)):
            v0, v2 = _vertex(q), _vertex(q2)
            if wv.sum() > 0:
                assert abs(v2.sum() - v0.sum()) < 1e-13 * max(1.0, np.abs(v0).sum())   # momentum conserved
                ex = wv * v0 + (v0 - wv * v0).sum() / wv.sum() * wv
                assert np.allclose(v2, ex, atol=1e-13)
            else:
                assert not q2.any()
            assert np.abs(v2[wv == 0]).max(initial=0) < 1e-15
    assert min(seen.values()) > 50, seen


def test_wetdry_tie_break_and_exact_threshold(O):
    h0 = 1e-3
    # vertex depth exactly H0 counts as dry (comparison is H > H0)
    hv = np.array([0.0, 1.0, 1.0])
    ze = np.array([0.0, 0.0, 0.0]); ze[0] = 0.0
    # zeta vertex values: choose modes so that zeta_v0 = H0, others 0 -> H = (H0, 1, 1)
    u = np.array([h0, 0.0, 0.0]); a = u.sum() / 3; ze = np.array([a, 0.5 * (u[2] - a), 0.5 * (u[1] - u[0])])
    wet, z2, x2, y2 = O.wetdry_elem(1, h0, hv, ze, [1.0, 0, 0], [0.0, 0, 0])
    assert wet == 1
    assert abs(_vertex(x2)[0]) < 1e-15 and abs(x2[0] - 1.0) < 1e-15   # v0 dry: its Q moved to v1, v2
    # p=2 pre-step: a quadratic dip below H0 at an interior point zeroes modes 3-5 of all variables
    ze6 = np.array([0.5, 0, 0, -2.0, 0, 0]); q6 = np.array([1.0, 0.1, 0.1, 0.2, 0.2, 0.2])
    wet, z2, x2, y2 = O.wetdry_elem(2, h0, np.array([1.0, 1.0, 1.0]), ze6, q6, q6)
    assert not z2[3:].any() and not x2[3:].any() and not y2[3:].any()
    wet, z2, x2, y2 = O.wetdry_elem(2, h0, np.array([9.0, 9.0, 9.0]), ze6, q6, q6)
    assert wet == 1 and np.array_equal(z2, ze6) and np.array_equal(x2, q6)


def test_set_state_initialises_wet_mask(O):
    w = c4(nqx=16, nqy=8)
    o = O.Oracle.from_workload(w)
    wet = o.get_wetdry()
    # initial film H0/2 on land, zeta = 0 over water: an element is dry iff its MEAN depth is <= H0 (case 3 of R-8);
    # with h_b linear in x and the film at H0/2 that is: mean of max(h_v, H0/2) over the vertices <= H0
    hv = w.bathy[w.mesh.tri]
    Hbar = np.maximum(hv, 0.5e-3).mean(axis=1)
    assert np.array_equal(wet == 0, Hbar <= 1e-3)
    assert abs((wet == 0).mean() - 0.2) < 0.05


# ------------------------------------------------------------------ wind
def test_det_exp_log_against_libm(O):
    rng = np.random.default_rng(2)
    for x in np.concatenate([rng.uniform(-50, 50, 500), [0.0, 1.0, -1.0, 1e-9, -700.5, 699.0]]):
        ex = math.exp(x) if x > -700 else 0.0
        assert abs(O.det_exp(x) - ex) <= 4e-16 * max(ex, 1e-300) * (1 + abs(x)) or ex == 0.0
    for x in np.concatenate([10 ** rng.uniform(-8, 8, 500), [1.0, 2.0, 0.5, math.sqrt(0.5), math.sqrt(2.0)]]):
        assert abs(O.det_log(x) - math.log(x)) <= 4e-16 * max(abs(math.log(x)), 1.0)


def test_holland_closed_forms(O):
    """At r = Rmax with f = 0 the gradient wind is sqrt(B dp / (rho_a e)) = 53.66 m/s for
    dp = 6000 Pa, B = 1.5, rho_a = 1.15 (V_max ~ 53.7 m/s); counter-clockwise;
    Garratt drag capped at 0.0035; stress = (rho_a/rho_0) C_d V W."""
    hol = dict(x0=0, y0=0, vx=0, vy=0, rmax=40e3, dp=6000.0, B=1.5, rho_air=1.15, rho_water=1025.0, f=0.0)
    tsx, tsy, V = O.holland_node(hol, 0.0, 0.0, 40e3, 0.0)
    vmax = math.sqrt(1.5 * 6000.0 / (1.15 * math.e))
    assert abs(vmax - 53.66) < 0.01 and abs(V - vmax) < 1e-12 * vmax
    assert abs(tsx) < 1e-18 and tsy > 0                        # east of the eye the wind blows north
    cd = min(0.0035, (0.75 + 0.067 * V) * 1e-3)
    assert cd == 0.0035
    assert abs(tsy - (1.15 / 1025.0) * cd * V * V) < 1e-15
    # generic point against libm pow/exp
    hol["f"] = 7e-5
    x, y = -13e3, 55e3
    tsx, tsy, V = O.holland_node(hol, 1e3, -2e3, x, y)
    dx, dy = x - 1e3, y + 2e3; r = math.hypot(dx, dy)
    xb = (40e3 / r) ** 1.5
    Vex = math.sqrt(1.5 / 1.15 * xb * 6000.0 * math.exp(-xb) + (r * 7e-5 / 2) ** 2) - r * 7e-5 / 2
    assert abs(V - Vex) < 1e-12 * Vex
    cd = min(0.0035, (0.75 + 0.067 * Vex) * 1e-3)
    k = 1.15 / 1025.0 * cd * Vex * Vex
    assert abs(tsx - k * (-dy / r)) < 1e-12 * k and abs(tsy - k * (dx / r)) < 1e-12 * k
    assert O.holland_node(hol, 0.0, 0.0, 0.5, 0.0) == (0.0, 0.0, 0.0)   # r < 1 m


def test_wind_moves_with_time_and_enters_rhs_only_when_wet(O):
    w = c4(nqx=16, nqy=8)
    o = O.Oracle.from_workload(w)
    r = o.eval_rhs()
    tau0 = o.get_wind()
    assert np.abs(tau0).max() > 1e-4
    wet = o.get_wetdry().astype(bool)
    o.set_wind_holland(None)
    r0 = o.eval_rhs()
    o.set_wind_holland(w.holland)
    dq = r[1][0] - r0[1][0]                      # wind contribution to d(mean Qx)/dt
    assert np.abs(dq[~wet]).max() == 0.0 and np.abs(dq[wet]).max() > 1e-6
    # mean of the nodal stress over the element (3-point rule is exact for linear tau)
    tbar = tau0[0][w.mesh.tri].mean(axis=1)
    assert np.allclose(dq[wet], tbar[wet], rtol=1e-9, atol=1e-15)
    o.step(3, w.dt)
    o.eval_rhs()
    assert np.abs(o.get_wind() - tau0).max() > 0


def test_nodal_output_pins(O):
    """orc_get_nodal (averaging the incident elements at every node): a continuous piecewise-linear field is
    returned exactly as its nodal values (every incident element has that value at the node); a discontinuous one
    gives the plain mean of the incident elements' vertex values (recomputed here with numpy's scatter-add from the
    closed-form vertex values u0 = a-b-c, u1 = a-b+c, u2 = a+2b of SURVEY.md 8(c.1)); interior nodes of the regular C1
    mesh see 6 elements, corner nodes 1 or 2."""
    from workloads import c1
    from workloads.configs import _modal
    w = c1(nq=6)
    m = w.mesh
    rng = np.random.default_rng(4)
    o = O.Oracle.from_workload(w)
    # (1) continuous linear field per variable
    f = [lambda x, y: 0.3 + 1e-4 * x - 2e-4 * y, lambda x, y: 1.0 + 3e-4 * x, lambda x, y: -2.0 + 5e-5 * y + 1e-4 * x]
    nodal = [fi(m.xy[:, 0], m.xy[:, 1]) for fi in f]
    st = [_modal(nv, m, 1) for nv in nodal]
    o.set_state(0.0, *st)
    for got, want in zip(o.get_nodal(), nodal):
        assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()
    # (2) random discontinuous modes against a numpy scatter-add of the closed-form vertex values
    st = [rng.uniform(-1, 1, (3, m.n_elem)) for _ in range(3)]
    o.set_state(0.0, *st)
    _, *st = o.get_state()          # (set_state runs the initial wet/dry pass; compare on what is stored)
    cnt = np.zeros(m.n_nodes); np.add.at(cnt, m.tri.ravel(), 1.0)
    assert cnt.max() == 6 and cnt.min() in (1, 2)
    for got, (a, b, c) in zip(o.get_nodal(), st):
        verts = np.stack([a - b - c, a - b + c, a + 2 * b], axis=1)      # [n_elem, 3]
        acc = np.zeros(m.n_nodes); np.add.at(acc, m.tri.ravel(), verts.ravel())
        assert np.abs(got - acc / cnt).max() <= 1e-14


def test_nodal_output_p2_uses_all_six_modes(O):
    """p = 2: vertex values from the closed-form table of SURVEY.md 8(c.1): phi00=(1,1,1), phi01=(-1,-1,2), phi10=(-1,1,0),
    phi02=(1,1,3), phi11=(1,-1,0), phi20=(1,1,0)."""
    from workloads import c2
    w = c2(nq=6, p=2, state="rest")
    m = w.mesh
    rng = np.random.default_rng(8)
    prm = dict(w.params); prm["wetdry"] = 0
    o = O.Oracle(prm, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    st = [rng.uniform(-1, 1, (6, m.n_elem)) for _ in range(3)]
    o.set_state(0.0, *st)
    V = np.array([[1, 1, 1], [-1, -1, 2], [-1, 1, 0], [1, 1, 3], [1, -1, 0], [1, 1, 0]], dtype=np.float64)   # [k][v]
    cnt = np.zeros(m.n_nodes); np.add.at(cnt, m.tri.ravel(), 1.0)
    for got, wv in zip(o.get_nodal(), st):
        verts = wv.T @ V                                             # [n_elem, 3]
        acc = np.zeros(m.n_nodes); np.add.at(acc, m.tri.ravel(), verts.ravel())
        assert np.abs(got - acc / cnt).max() <= 1e-13
