"""Pins for the Roe numerical flux ("Local Lax-Friedrichs or Roe"; R-17).
Expected values: the physical flux (consistency, upwinding in supercritical flow), the textbook matrix form
1/2 (F+ + F-).n - 1/2 |A~| (w- - w+) with |A~| from numpy's eigen-decomposition of the Roe matrix in the x-y frame,
exact preservation of a stationary contact (shear) discontinuity, and -- through the model -- lake at rest, mass
conservation and the seiche convergence order."""
import math

import numpy as np
import pytest

from helpers import G, l2_project, llf_xy, phys_flux, small_mesh
from workloads import c2, default_params
from workloads.mesh import rect_mesh

H0 = 1e-3


def roe_matrix_form(wp, wm, h, n):
    """Textbook Roe flux in the x-y frame with conserved variables (H, Qx, Qy) (same bed on both sides)."""
    Hp, Hm = wp[0] + h, wm[0] + h
    up, vp, um, vm = wp[1] / Hp, wp[2] / Hp, wm[1] / Hm, wm[2] / Hm
    sp, sm = math.sqrt(Hp), math.sqrt(Hm)
    u = (sp * up + sm * um) / (sp + sm)
    v = (sp * vp + sm * vm) / (sp + sm)
    c2_ = G * 0.5 * (Hp + Hm)
    nx, ny = n
    A = np.array([[0.0, nx, ny],
                  [(c2_ - u * u) * nx - u * v * ny, 2 * u * nx + v * ny, u * ny],
                  [-u * v * nx + (c2_ - v * v) * ny, v * nx, u * nx + 2 * v * ny]])
    lam, R = np.linalg.eig(A)
    absA = (R * np.abs(lam)) @ np.linalg.inv(R)
    Fxp, Fyp = phys_flux(*[np.float64(x) for x in wp], h, H0)
    Fxm, Fym = phys_flux(*[np.float64(x) for x in wm], h, H0)
    dw = np.array(wm, dtype=float) - np.array(wp, dtype=float)
    return 0.5 * ((Fxp + Fxm) * nx + (Fyp + Fym) * ny) - 0.5 * (absA.real @ dw)


def _states(rng, sub=True):
    th = rng.uniform(0, 2 * np.pi); n = (math.cos(th), math.sin(th))
    h = rng.uniform(2.0, 50.0)
    sc = 3.0 if sub else 1.0
    wp = [rng.uniform(-0.4, 1), rng.uniform(-5, 5) * sc, rng.uniform(-5, 5) * sc]
    wm = [rng.uniform(-0.4, 1), rng.uniform(-5, 5) * sc, rng.uniform(-5, 5) * sc]
    return n, h, wp, wm


def test_roe_consistency_and_matrix_form(O):
    rng = np.random.default_rng(0)
    for _ in range(200):
        n, h, wp, wm = _states(rng)
        f = O.roe_flux(G, H0, n[0], n[1], h, wp, wp)
        Fx, Fy = phys_flux(*[np.float64(x) for x in wp], h, H0)
        assert np.allclose(f, Fx * n[0] + Fy * n[1], rtol=1e-12, atol=1e-11)          # F^(w, w) = F(w).n
        f = O.roe_flux(G, H0, n[0], n[1], h, wp, wm)
        ex = roe_matrix_form(wp, wm, h, n)
        assert np.allclose(f, ex, rtol=1e-10, atol=1e-9 * max(1.0, np.abs(ex).max()))


def test_roe_upwinds_in_supercritical_flow(O):
    """All three Roe speeds of one sign: the flux is the physical flux of the upwind trace (the linearisation is exact:
    F(w-) - F(w+) = sum lambda_k a_k r_k).  LLF does not have this property."""
    rng = np.random.default_rng(1)
    n_pos = n_neg = 0
    for _ in range(400):
        th = rng.uniform(0, 2 * np.pi); n = (math.cos(th), math.sin(th))
        h = rng.uniform(1.0, 3.0)
        sgn = 1.0 if rng.uniform() < 0.5 else -1.0
        qn = sgn * rng.uniform(25.0, 40.0, 2)                    # |u_n| ~ 10-30 m/s against c ~ 4-6 m/s
        qt = rng.uniform(-5, 5, 2)
        wp = [rng.uniform(-0.2, 0.4), qn[0] * n[0] - qt[0] * n[1], qn[0] * n[1] + qt[0] * n[0]]
        wm = [rng.uniform(-0.2, 0.4), qn[1] * n[0] - qt[1] * n[1], qn[1] * n[1] + qt[1] * n[0]]
        f = O.roe_flux(G, H0, n[0], n[1], h, wp, wm)
        up = wp if sgn > 0 else wm
        Fx, Fy = phys_flux(*[np.float64(x) for x in up], h, H0)
        ex = Fx * n[0] + Fy * n[1]
        assert np.allclose(f, ex, rtol=1e-11, atol=1e-9), (sgn, f, ex)
        n_pos += sgn > 0; n_neg += sgn < 0
        lf = O.llf_flux(G, H0, n[0], n[1], h, wp, wm)
        assert np.abs(lf - ex).max() > 1e-3 * np.abs(ex).max() or np.allclose(wp, wm)
    assert n_pos > 100 and n_neg > 100


def test_roe_preserves_a_stationary_contact_exactly(O):
    """Equal depths, no normal flow, a jump in the tangential momentum only: mass flux 0, tangential momentum flux 0,
    normal momentum flux = pressure -- exactly; LLF smears the shear (-lambda/2 dq_t)."""
    rng = np.random.default_rng(2)
    for _ in range(50):
        th = rng.uniform(0, 2 * np.pi); n = (math.cos(th), math.sin(th))
        h, z = rng.uniform(1, 30), rng.uniform(-0.3, 0.5)
        qtp, qtm = rng.uniform(-5, 5, 2)
        wp = [z, -qtp * n[1], qtp * n[0]]
        wm = [z, -qtm * n[1], qtm * n[0]]
        f = O.roe_flux(G, H0, n[0], n[1], h, wp, wm)
        P = G * z * (0.5 * z + h)
        scale = abs(P) + 1.0
        assert abs(f[0]) <= 1e-15 * 10
        assert abs(f[1] - P * n[0]) <= 1e-13 * scale and abs(f[2] - P * n[1]) <= 1e-13 * scale
        lf = O.llf_flux(G, H0, n[0], n[1], h, wp, wm)
        assert np.hypot(lf[1] - P * n[0], lf[2] - P * n[1]) > 0.1 * abs(qtm - qtp)


def test_roe_antisymmetry_bitwise_wall_and_ocean(O):
    rng = np.random.default_rng(3)
    for _ in range(200):
        n, h, wp, wm = _states(rng)
        f1 = O.roe_flux(G, H0, n[0], n[1], h, wp, wm)
        f2 = O.roe_flux(G, H0, -n[0], -n[1], h, wm, wp)
        assert np.array_equal(f1, -f2)
        fw = O.roe_flux(G, H0, n[0], n[1], h, wp, [9, 9, 9], bc=1)
        assert fw[0] == 0.0                                          # wall: exactly no mass flux
        qn = wp[1] * n[0] + wp[2] * n[1]
        mirror = [wp[0], wp[1] - 2 * qn * n[0], wp[2] - 2 * qn * n[1]]
        assert np.allclose(fw, roe_matrix_form(wp, mirror, h, n), rtol=1e-10, atol=1e-9 * max(1.0, np.abs(fw).max()))
        fo = O.roe_flux(G, H0, n[0], n[1], h, wp, [9, 9, 9], bc=2, zeta_b=0.37)
        assert np.allclose(fo, roe_matrix_form(wp, [0.37, wp[1], wp[2]], h, n), rtol=1e-10, atol=1e-9 * max(1.0, np.abs(fo).max()))


def test_roe_depth_floor(O):
    f = O.roe_flux(G, H0, 1.0, 0.0, 0.0, [1e-6, 1e-5, 0.0], [2e-6, -1e-5, 0.0])
    assert np.all(np.isfinite(f))


def _oracle(O, mesh, bathy, **kw):
    prm = default_params(**kw)
    return O.Oracle(prm, mesh.xy, bathy, mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)


@pytest.mark.parametrize("p", [1, 2])
def test_roe_in_the_model_lake_at_rest_and_conservation(O, p):
    w = c2(nq=12, p=p, state="rest")
    prm = dict(w.params); prm["flux"] = 1
    m = w.mesh
    o = O.Oracle(prm, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    o.set_state(0.0, w.ze, w.qx, w.qy)
    r, s = o.eval_rhs(with_scale=True)
    for c in range(3):
        assert np.abs(r[c]).max() <= 1e-13 * max(s[c].max(), 1.0)      # well balanced with Roe too
    w = c2(nq=12, p=p, state="hump")
    o = O.Oracle(prm, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    o.set_state(0.0, w.ze, w.qx, w.qy)
    area = o.get_geometry()[0]
    m0 = float((area * w.ze[0]).sum())
    o.step(40, w.dt)
    _, ze, qx, qy = o.get_state()
    assert np.isfinite(ze).all() and np.abs(qx).max() > 1e-3
    assert abs(float((area * ze[0]).sum()) - m0) < 1e-13 * 1e9          # closed walls: mass to round-off
    # and the result differs from the LLF run (the switch is wired)
    o2 = O.Oracle.from_workload(w); o2.step(40, w.dt)
    assert np.abs(o2.get_state()[1] - ze).max() > 1e-8


@pytest.mark.parametrize("p", [1, 2])
def test_roe_seiche_convergence_order(O, p):
    """The textbook seiche (period 2019 s) with the Roe flux: order ~ p + 1, as with LLF."""
    L, H, amp, t_end = 10_000.0, 10.0, 1e-4, 300.0
    k = math.pi / L
    om = k * math.sqrt(G * H)
    errs = []
    for nq in ((8, 16, 32) if p == 1 else (4, 8, 16)):
        mesh = rect_mesh(nq, nq, L, L, diag="same")
        o = _oracle(O, mesh, np.full(mesh.n_nodes, H), p=p, rk_order=3, flux=1)
        ze0 = l2_project(O, mesh, lambda x, y: amp * np.cos(k * x), p)
        o.set_state(0.0, ze0, 0 * ze0, 0 * ze0)
        dt = 0.1 * (L / nq) / ((2 * p + 1) * math.sqrt(G * H))
        n = int(math.ceil(t_end / dt)); dt = t_end / n
        o.step(n, dt)
        t, ze, _, _ = o.get_state()
        zex = l2_project(O, mesh, lambda x, y: amp * np.cos(k * x) * math.cos(om * t), p)
        Mref = np.array([2.0, 1.0, 1 / 3, 2 / 3, 2 / 9, 2 / 15])[:ze.shape[0], None]
        l2 = lambda a: math.sqrt(float((a * a * Mref).sum()))
        errs.append(l2(ze - zex) / l2(zex))
    o1, o2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert o2 > p + 0.6 and o1 > p + 0.3, errs
