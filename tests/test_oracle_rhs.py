"""Pins for the oracle's numerical flux and RHS (eqs (1)-(3), (6)-(10), Algs 1-3).
SURVEY.md §8(c.5): consistency / antisymmetry / wall flux; constant state; lake at rest;
rotation equivariance; brute force with dense mass solve on tiny meshes."""
import numpy as np
import pytest

from helpers import (G, brute_force_rhs, l2_project, llf_xy, phys_flux, small_mesh, two_element_mesh)
from workloads import c2, default_params
from workloads.mesh import make_mesh, vertex_to_modal_p1


def make_oracle(O, mesh, bathy, **kw):
    prm = default_params(**kw)
    return O.Oracle(prm, mesh.xy, bathy, mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)


# ------------------------------------------------------------------ LLF flux
def test_llf_consistency(O):
    """F^(w, w) = F(w).n  (eqs (7)-(9))."""
    rng = np.random.default_rng(0)
    for _ in range(50):
        th = rng.uniform(0, 2 * np.pi); n = (np.cos(th), np.sin(th))
        h = rng.uniform(1, 50); w = (rng.uniform(-1, 1), rng.uniform(-5, 5), rng.uniform(-5, 5))
        f = O.llf_flux(G, 1e-3, n[0], n[1], h, w, w)
        Fx, Fy = phys_flux(*[np.float64(x) for x in w], h, 1e-3)
        ex = Fx * n[0] + Fy * n[1]
        assert np.allclose(f, ex, rtol=1e-13, atol=1e-12)


def test_llf_matches_xy_frame_formula(O):
    """Rotated-frame implementation == textbook x-y frame LLF on discontinuous states."""
    rng = np.random.default_rng(1)
    for _ in range(100):
        th = rng.uniform(0, 2 * np.pi); n = (np.cos(th), np.sin(th))
        h = rng.uniform(0.5, 50)
        wp = [rng.uniform(-0.4, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        wm = [rng.uniform(-0.4, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        f = O.llf_flux(G, 1e-3, n[0], n[1], h, wp, wm)
        ex = llf_xy([np.float64(x) for x in wp], [np.float64(x) for x in wm], h, n, 1e-3)
        assert np.allclose(f, ex, rtol=1e-12, atol=1e-11)


def test_llf_antisymmetry_bitwise(O):
    """(w+, w-, n) -> (w-, w+, -n) flips the sign exactly."""
    rng = np.random.default_rng(2)
    for _ in range(100):
        th = rng.uniform(0, 2 * np.pi); n = (np.cos(th), np.sin(th))
        h = rng.uniform(0.5, 50)
        wp = [rng.uniform(-0.4, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        wm = [rng.uniform(-0.4, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        f1 = O.llf_flux(G, 1e-3, n[0], n[1], h, wp, wm)
        f2 = O.llf_flux(G, 1e-3, -n[0], -n[1], h, wm, wp)
        assert np.array_equal(f1, -f2)


def test_wall_mass_flux_exactly_zero_and_ocean_state(O):
    rng = np.random.default_rng(3)
    for _ in range(100):
        th = rng.uniform(0, 2 * np.pi); n = (np.cos(th), np.sin(th))
        h = rng.uniform(0.5, 50)
        wp = [rng.uniform(-0.4, 1), rng.uniform(-5, 5), rng.uniform(-5, 5)]
        f = O.llf_flux(G, 1e-3, n[0], n[1], h, wp, [9, 9, 9], bc=1)
        assert f[0] == 0.0
        # momentum flux of a wall = mirror state in the x-y formula
        qn = wp[1] * n[0] + wp[2] * n[1]
        wm = [wp[0], wp[1] - 2 * qn * n[0], wp[2] - 2 * qn * n[1]]
        ex = llf_xy([np.float64(x) for x in wp], [np.float64(x) for x in wm], h, n, 1e-3)
        assert np.allclose(f[1:], ex[1:], rtol=1e-12, atol=1e-11)
        fo = O.llf_flux(G, 1e-3, n[0], n[1], h, wp, [9, 9, 9], bc=2, zeta_b=0.37)
        exo = llf_xy([np.float64(x) for x in wp], [np.float64(0.37), np.float64(wp[1]), np.float64(wp[2])], h, n, 1e-3)
        assert np.allclose(fo, exo, rtol=1e-12, atol=1e-11)


def test_depth_floor_in_flux(O):
    """H_c = max(H, H0): a nearly dry trace gives finite flux, velocity computed with H0."""
    f = O.llf_flux(G, 1e-3, 1.0, 0.0, 0.0, [1e-6, 1e-5, 0.0], [1e-6, 1e-5, 0.0])
    assert np.all(np.isfinite(f))
    assert abs(f[1] - (1e-5 * 1e-5 / 1e-3 + 0.5 * G * 1e-12)) < 1e-18


# ------------------------------------------------------------------ RHS invariants
@pytest.mark.parametrize("p", [1, 2, 3])
def test_constant_state_flat_bottom_rhs_zero_in_interior(O, p):
    """A constant state (zeta, Qx, Qy) on a flat bottom is preserved by every element that has
    no wall edge (walls reflect the momentum)."""
    mesh = small_mesh(nq=5)
    ndof = (p + 1) * (p + 2) // 2
    o = make_oracle(O, mesh, np.full(mesh.n_nodes, 12.0), p=p, cf=0.0)
    st = np.zeros((3, ndof, mesh.n_elem)); st[0, 0] = 0.7; st[1, 0] = 3.0; st[2, 0] = -2.0
    o.set_state(0.0, *st)
    r, s = o.eval_rhs(with_scale=True)
    has_wall = (mesh.edge_bc[mesh.elem_edge] != 0).any(axis=1)
    assert (~has_wall).sum() > 10
    for c in range(3):
        assert np.abs(r[c][:, ~has_wall]).max() <= 1e-13 * s[c].max()
    assert max(np.abs(r[c][:, has_wall]).max() for c in (1, 2)) > 1e-3     # walls do act


@pytest.mark.parametrize("p", [1, 2, 3])
def test_lake_at_rest_variable_bathymetry(O, p):
    """Well-balancedness: zeta = const, Q = 0 over variable continuous piecewise-linear h_b
    gives RHS = 0 (to round-off relative to the size of the cancelling terms) and the state
    does not move in N steps."""
    w = c2(nq=12, p=p, state="rest")
    o = O.Oracle.from_workload(w)
    r, s = o.eval_rhs(with_scale=True)
    for c in range(3):
        assert np.abs(r[c]).max() <= 1e-13 * max(s[c].max(), 1.0)
    o.step(25, w.dt)
    _, ze, qx, qy = o.get_state()
    assert np.abs(ze[0] - 0.3).max() < 1e-12 and np.abs(ze[1:]).max() < 1e-12
    assert max(np.abs(qx).max(), np.abs(qy).max()) < 1e-11


def test_lake_at_rest_with_ocean_boundary_at_same_level(O):
    mesh = small_mesh(nq=4, ocean=True)
    rng = np.random.default_rng(5)
    bathy = 20.0 + 5.0 * rng.uniform(-1, 1, mesh.n_nodes)
    o = make_oracle(O, mesh, bathy, p=1)
    ze = np.zeros((3, mesh.n_elem)); ze[0] = 0.25
    o.set_state(0.0, ze, 0 * ze, 0 * ze)
    o.set_tide(0.25, 0.0, np.pi / 2)          # zeta_b = 0.25 sin(pi/2) = 0.25
    r, s = o.eval_rhs(with_scale=True)
    for c in range(3):
        assert np.abs(r[c]).max() <= 1e-13 * max(s[c].max(), 1.0)


@pytest.mark.parametrize("p", [1, 2, 3])
def test_rotation_equivariance(O, p):
    """Rotating mesh and momentum by 90 degrees rotates the RHS: (x,y)->(-y,x), (Qx,Qy)->(-Qy,Qx)."""
    mesh = small_mesh(nq=3, permute=False)
    rng = np.random.default_rng(11)
    bathy = 15.0 + 3.0 * rng.uniform(-1, 1, mesh.n_nodes)
    ndof = (p + 1) * (p + 2) // 2
    st = 0.1 * rng.uniform(-1, 1, (3, ndof, mesh.n_elem)); st[1:] *= 20.0
    kw = dict(p=p, cf=0.003)       # Coriolis off: it is rotation-equivariant too, but keep the pin simple
    o1 = make_oracle(O, mesh, bathy, **kw)
    o1.set_state(0.0, *st)
    r1 = o1.eval_rhs()
    xy2 = np.stack([-mesh.xy[:, 1], mesh.xy[:, 0]], axis=1)
    mesh2 = make_mesh(xy2, mesh.tri)     # same connectivity; the modal coefficients are invariant
    assert np.array_equal(mesh2.elem_edge, mesh.elem_edge)
    o2 = make_oracle(O, mesh2, bathy, **kw)
    o2.set_state(0.0, st[0], -st[2], st[1])
    r2 = o2.eval_rhs()
    scale = max(np.abs(r1[c]).max() for c in range(3))
    assert np.abs(r2[0] - r1[0]).max() < 1e-12 * scale
    assert np.abs(r2[1] - (-r1[2])).max() < 1e-12 * scale
    assert np.abs(r2[2] - r1[1]).max() < 1e-12 * scale


# ------------------------------------------------------------------ brute force
def _smooth_state(O, mesh, p, kind, seed=3):
    rng = np.random.default_rng(seed)
    if kind == "poly_exact":
        # Q = 0 and a continuous LINEAR zeta: P = g zeta (zeta/2 + h_b) has degree 2, so every
        # integrand is a polynomial the oracle's rules integrate exactly (volume: 2 + (p-1) <= 2p,
        # edge: 2 + p <= 2p+1)
        fz = lambda x, y: 0.3 + 2e-4 * x - 1e-4 * y
        W = [l2_project(O, mesh, fz, p), None, None]
        W[1] = np.zeros_like(W[0]); W[2] = np.zeros_like(W[0])
        return W
    if kind == "continuity_exact":
        # continuous zeta (linear) and continuous Q of full degree p: the continuity row
        # int Q.grad(phi) - oint Q.n phi is integrated exactly and has no LLF jump term
        fz = lambda x, y: 0.3 + 2e-4 * x - 1e-4 * y
        if p == 1:
            fx = lambda x, y: 1.0 + 2e-3 * x - 1e-3 * y
            fy = lambda x, y: -0.5 + 1e-3 * x + 3e-3 * y
        elif p == 2:
            fx = lambda x, y: 1.0 + 2e-3 * x - 1e-3 * y + 1e-6 * x * y - 2e-6 * x * x
            fy = lambda x, y: -0.5 + 1e-3 * x + 3e-3 * y + 2e-6 * y * y - 1e-6 * x * y
        else:
            fx = lambda x, y: 1.0 + 2e-3 * x - 1e-3 * y + 1e-6 * x * y - 2e-6 * x * x + 3e-9 * x * x * x - 2e-9 * x * y * y
            fy = lambda x, y: -0.5 + 1e-3 * x + 3e-3 * y + 2e-6 * y * y - 1e-6 * x * y - 1e-9 * y * y * y + 4e-9 * x * x * y
        return [l2_project(O, mesh, f, p) for f in (fz, fx, fy)]
    # generic: discontinuous, all three variables, mild amplitude
    ndof = (p + 1) * (p + 2) // 2
    W = [l2_project(O, mesh, lambda x, y: 0.2 * np.sin(2e-3 * x) * np.cos(1e-3 * y), p),
         l2_project(O, mesh, lambda x, y: 1.5 * np.cos(1e-3 * x + 2e-3 * y), p),
         l2_project(O, mesh, lambda x, y: -1.0 * np.sin(2e-3 * x - 1e-3 * y), p)]
    for c in range(3):
        W[c] = W[c] + (0.02 if c == 0 else 0.1) * rng.uniform(-1, 1, (ndof, mesh.n_elem)) * (np.arange(ndof)[:, None] < 3)
    return W


@pytest.mark.parametrize("p", [1, 2, 3])
@pytest.mark.parametrize("which", ["two", "eight"])
def test_bruteforce_polynomial_exact_case(O, p, which):
    """Where the oracle's quadrature is exact, its RHS equals the weak form (3) integrated
    with a 12x12 / 10-point rule and solved with a DENSE mass matrix, to round-off."""
    mesh = two_element_mesh() if which == "two" else small_mesh(nq=2, L=1000.0)
    rng = np.random.default_rng(4)
    bathy = 10.0 + 2.0 * rng.uniform(-1, 1, mesh.n_nodes)
    W = _smooth_state(O, mesh, p, "poly_exact")
    o = make_oracle(O, mesh, bathy, p=p)
    o.set_state(0.0, *W)
    r = np.stack(o.eval_rhs())
    bf = brute_force_rhs(O, mesh, bathy, p, *W)
    assert np.abs(bf[1:]).max() > 1e-4
    assert np.abs(r - bf).max() < 1e-11 * max(1.0, np.abs(bf).max())


@pytest.mark.parametrize("p", [1, 2, 3])
def test_bruteforce_generic_state_within_quadrature_error(O, p):
    """Discontinuous state with momentum, friction, Coriolis, an ocean boundary: the oracle
    differs from the exactly integrated weak form only by its quadrature error (non-polynomial
    Q^2/H, |Q|/H^2 and lambda), which is small for this mild state; a dropped term, wrong sign
    or transposed index would be O(1)."""
    mesh = small_mesh(nq=2, L=1000.0, ocean=True)
    rng = np.random.default_rng(8)
    bathy = 10.0 + 2.0 * rng.uniform(-1, 1, mesh.n_nodes)
    W = _smooth_state(O, mesh, p, "generic")
    o = make_oracle(O, mesh, bathy, p=p, cf=0.0025, coriolis_f=1e-2)
    o.set_tide(0.1, 0.0, np.pi / 2)
    o.set_state(0.0, *W)
    r = np.stack(o.eval_rhs())
    bf = brute_force_rhs(O, mesh, bathy, p, *W, cf=0.0025, fcor=1e-2, zeta_b=0.1)
    for c in range(3):
        sc = np.abs(bf[c]).max()
        assert sc > 1e-4
        assert np.abs(r[c] - bf[c]).max() < (2e-3 if p == 1 else 2e-4) * sc


@pytest.mark.parametrize("p", [1, 2, 3])
def test_bruteforce_continuity_row_exact_with_full_degree_momentum(O, p):
    mesh = small_mesh(nq=2, L=1000.0)
    bathy = np.full(mesh.n_nodes, 10.0)
    W = _smooth_state(O, mesh, p, "continuity_exact")
    assert p == 1 or np.abs(W[1][3:6]).max() > 1e-3         # quadratic state modes are exercised
    assert p < 3 or np.abs(W[1][6:]).min(axis=1).max() > 0 and np.abs(W[1][6:]).max() > 1e-3   # ... and the cubic ones
    o = make_oracle(O, mesh, bathy, p=p)
    o.set_state(0.0, *W)
    r = np.stack(o.eval_rhs())
    bf = brute_force_rhs(O, mesh, bathy, p, *W)
    assert np.abs(bf[0]).max() > 1e-4
    assert np.abs(r[0] - bf[0]).max() < 1e-11 * max(1.0, np.abs(bf[0]).max())
    for c in (1, 2):
        assert np.abs(r[c] - bf[c]).max() < 2e-3 * np.abs(bf[c]).max()


def test_flux_buffer_and_gather_sign_convention(O):
    """Per-edge flux buffer: F^ is the flux leaving e+ (n from e+ to e-); swapping which side is
    e+ (a renumbering the generator controls) must not change the RHS."""
    mesh = small_mesh(nq=3)
    rng = np.random.default_rng(9)
    bathy = 10.0 + rng.uniform(-1, 1, mesh.n_nodes)
    st = 0.1 * rng.uniform(-1, 1, (3, 3, mesh.n_elem)); st[1:] *= 10
    o = make_oracle(O, mesh, bathy, p=1)
    o.set_state(0.0, *st)
    r1 = np.stack(o.eval_rhs())
    f1 = o.get_flux()
    ee, el = mesh.edge_elem.copy(), mesh.edge_local.copy()
    inter = ee[:, 1] >= 0
    ee[inter] = ee[inter][:, ::-1]; el[inter] = el[inter][:, ::-1]
    o2 = O.Oracle(default_params(p=1), mesh.xy, bathy, mesh.tri, ee, el, mesh.edge_bc, mesh.elem_edge)
    o2.set_state(0.0, *st)
    r2 = np.stack(o2.eval_rhs())
    f2 = o2.get_flux()
    assert np.array_equal(f2[:, ::-1, inter], -f1[:, :, inter])      # antisymmetric, points reversed
    assert np.abs(r1 - r2).max() <= 1e-13 * np.abs(r1).max()
