"""Pins for the atmospheric-pressure-gradient and rain sources ("R the mass
source term such as rain", :65 forcings, :326 "Wind forcing and pressure calculations (WIND)"; R-15, R-16).
Expected values come from closed forms (Holland 1980 pressure profile with libm, the inverse-barometer balance,
integral of a constant source), never from the oracle's intermediates."""
import math

import numpy as np
import pytest

from helpers import G, small_mesh
from workloads import default_params
from workloads.configs import _modal
from workloads.mesh import rect_mesh

HOL = dict(x0=300.0, y0=-200.0, vx=0.0, vy=0.0, rmax=4000.0, dp=6000.0, B=1.5, rho_air=1.15, rho_water=1025.0, f=5e-5)


def make_oracle(O, mesh, bathy, **kw):
    prm = default_params(**kw)
    return O.Oracle(prm, mesh.xy, bathy, mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)


def test_holland_pressure_profile_closed_form(O):
    """eta_p(r) = -(dp/(rho_0 g)) (1 - exp(-(R/r)^B)): -dp/(rho_0 g) = -0.5967 m in the eye, -(1 - 1/e) of it at
    r = R, -> 0 far away; the stress outputs are those of orc_holland_node (same bits)."""
    full = HOL["dp"] / (HOL["rho_water"] * G)
    assert abs(full - 0.59672) < 1e-4
    for (x, y) in [(4300.0, -200.0), (300.0, 3800.0), (-9000.0, 12000.0), (300.5, -200.0), (1e6, 2e6)]:
        tsx, tsy, V, ep = O.holland_node_p(HOL, G, HOL["x0"], HOL["y0"], x, y)
        r = math.hypot(x - HOL["x0"], y - HOL["y0"])
        want = -full if r < 1.0 else -full * (1.0 - math.exp(-(HOL["rmax"] / r) ** HOL["B"]))
        assert abs(ep - want) <= 1e-13 * full
        assert (tsx, tsy, V) == O.holland_node(HOL, HOL["x0"], HOL["y0"], x, y)
    _, _, _, ep = O.holland_node_p(HOL, G, HOL["x0"], HOL["y0"], HOL["x0"] + HOL["rmax"], HOL["y0"])
    assert abs(ep + full * (1.0 - math.exp(-1.0))) < 1e-13


@pytest.mark.parametrize("p", [1, 2])
def test_inverse_barometer_is_a_discrete_steady_state(O, p):
    """zeta = -eta_p (the nodal pressure anomaly, element-wise linear, continuous), Q = 0, variable bathymetry, stress
    off: -g H grad(eta_p) balances g H grad(zeta) to ROUND-OFF, not just to quadrature error -- the same exactness
    argument as lake at rest (every integrand is a polynomial the rules integrate exactly) -- and the state does not
    move.  A wrong sign, a missing H, or H_c instead of H in the source leaves an O(1) residual."""
    mesh = small_mesh(nq=6, L=12000.0, seed=12)
    rng = np.random.default_rng(12)
    bathy = 30.0 + 8.0 * rng.uniform(-1, 1, mesh.n_nodes)
    o = make_oracle(O, mesh, bathy, p=p, rk_order=3)
    o.set_wind_holland(HOL)
    o.set_wind_forcing(stress=False, pressure=True)
    z0 = np.zeros(((p + 1) * (p + 2) // 2, mesh.n_elem))
    o.set_state(0.0, z0, z0, z0)
    o.eval_rhs()                                    # evaluates the nodal fields
    ep = o.get_pressure()
    full = HOL["dp"] / (HOL["rho_water"] * G)
    assert ep.min() < -0.4 * full and ep.max() > -0.3 * full    # a real gradient across the mesh
    # closed form at the nodes
    r = np.hypot(mesh.xy[:, 0] - HOL["x0"], mesh.xy[:, 1] - HOL["y0"])
    assert np.abs(ep + full * (1.0 - np.exp(-(HOL["rmax"] / r) ** HOL["B"]))).max() < 1e-13
    ze = _modal(-ep, mesh, p)
    o.set_state(0.0, ze, 0 * ze, 0 * ze)
    r_ib, s_ib = o.eval_rhs(with_scale=True)
    for c in range(3):
        assert np.abs(r_ib[c]).max() <= 1e-13 * max(s_ib[c].max(), 1.0)
    # without the balancing elevation the source is O(g H grad eta_p): the pin has teeth
    o.set_state(0.0, z0, z0, z0)
    r_flat = o.eval_rhs()
    assert np.abs(r_flat[1]).max() > 1e-3
    # and the balanced state stays put
    o.set_state(0.0, ze, 0 * ze, 0 * ze)
    o.step(20, 2.0)
    _, z1, qx1, qy1 = o.get_state()
    assert np.abs(z1 - ze).max() < 1e-12 and max(np.abs(qx1).max(), np.abs(qy1).max()) < 1e-10


def test_pressure_gradient_source_magnitude_and_wet_gate(O):
    """Flat water of depth h over a flat bed: d(mean Q)/dt = -g h grad(eta_p) with grad(eta_p) the gradient of the
    element's linear interpolant of the nodal anomaly (numpy, from the vertex coordinates); no contribution to the
    continuity equation; none in an element flagged dry; none with the switch off."""
    mesh = rect_mesh(5, 4, 10000.0, 8000.0, diag="same")
    h = 15.0
    o = make_oracle(O, mesh, np.full(mesh.n_nodes, h), p=1)
    o.set_wind_holland(HOL)
    z0 = np.zeros((3, mesh.n_elem))
    wet = np.ones(mesh.n_elem, dtype=np.uint8); wet[7] = 0
    o.set_state_raw(0.0, z0, z0, z0, wet)
    o.set_wind_forcing(stress=False, pressure=False)
    r_off = np.stack(o.eval_rhs())
    o.set_wind_forcing(stress=False, pressure=True)
    r_on = np.stack(o.eval_rhs())
    d = r_on - r_off
    ep = o.get_pressure()
    X = mesh.xy[mesh.tri]                                  # [ne, 3, 2]
    P = ep[mesh.tri]
    d1, d2 = X[:, 1] - X[:, 0], X[:, 2] - X[:, 0]
    det = d1[:, 0] * d2[:, 1] - d2[:, 0] * d1[:, 1]
    gx = ((P[:, 1] - P[:, 0]) * d2[:, 1] - (P[:, 2] - P[:, 0]) * d1[:, 1]) / det
    gy = (-(P[:, 1] - P[:, 0]) * d2[:, 0] + (P[:, 2] - P[:, 0]) * d1[:, 0]) / det
    live = wet == 1
    sc = np.abs(G * h * gx).max()
    assert sc > 1e-4
    assert np.abs(d[1, 0, live] + G * h * gx[live]).max() <= 1e-12 * sc
    assert np.abs(d[2, 0, live] + G * h * gy[live]).max() <= 1e-12 * sc
    assert not d[0].any() and not d[:, :, 7].any()
    assert np.abs(d[1:, 1:][:, :, live]).max() <= 1e-12 * sc      # H is constant: no projection on the linear modes
    # the depth in the source is the actual H = zeta + h_b, not the floored H_c: a film of 0.3 H0 in an element that is
    # still flagged wet feels 0.3 H0 of the force, not H0 of it
    h0 = 1e-3
    zt = z0.copy(); zt[0, 11] = 0.3 * h0 - h
    wet2 = np.ones(mesh.n_elem, dtype=np.uint8)
    o.set_state_raw(0.0, zt, z0, z0, wet2)
    o.set_wind_forcing(stress=False, pressure=False)
    ra = np.stack(o.eval_rhs())
    o.set_wind_forcing(stress=False, pressure=True)
    rb = np.stack(o.eval_rhs())
    assert abs((rb - ra)[1, 0, 11] + G * 0.3 * h0 * gx[11]) <= 1e-6 * G * h0 * abs(gx[11])   # (differences of O(g h^2 L/A) terms: round-off ~1e-9 of this)


@pytest.mark.parametrize("p", [1, 2])
def test_rain_is_a_uniform_mass_source(O, p):
    """S_zeta = R: d(zeta_00)/dt = R exactly in every element, wet or dry, nothing on the other modes
    beyond round-off, nothing on the momentum equations; with closed walls the total mass grows by R t |Omega|."""
    mesh = small_mesh(nq=5, L=2000.0, seed=5)
    rng = np.random.default_rng(5)
    bathy = 6.0 + rng.uniform(-1, 1, mesh.n_nodes)
    nd = (p + 1) * (p + 2) // 2
    o = make_oracle(O, mesh, bathy, p=p, wetdry=1, limiter=1)
    st = np.zeros((3, nd, mesh.n_elem)); st[0, 0] = 0.2
    st[0, 0, 3] = -bathy[mesh.tri[3]].mean() + 2e-4             # one dry element
    o.set_state(0.0, *st)
    assert o.get_wetdry()[3] == 0
    r0 = np.stack(o.eval_rhs())
    R = 2.5e-5                                                   # 90 mm/h
    o.set_rain(R)
    r1 = np.stack(o.eval_rhs())
    d = r1 - r0
    assert np.abs(d[0, 0] - R).max() <= 1e-16 * 1 + 4e-16 * np.abs(r0[0, 0]).max() + 1e-20
    assert np.abs(d[0, 1:]).max() <= 1e-17 + 4e-16 * np.abs(r0[0]).max()
    assert not d[1:].any()
    area = o.get_geometry()[0]
    _, z, _, _ = o.get_state()
    m0 = float((area * z[0]).sum())
    nsteps, dt = 40, 0.5
    o.step(nsteps, dt)
    _, z, _, _ = o.get_state()
    gain = float((area * z[0]).sum()) - m0
    assert abs(gain - R * nsteps * dt * area.sum()) <= 1e-12 * abs(m0)
