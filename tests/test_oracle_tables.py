"""Pins for the oracle's tables: Dubiner basis, reference mass, quadrature, geometry.
PAPER.md:97-107 (eq. (4), diagonal mass matrix, quadrature); SURVEY.md §8(c.5)."""
from itertools import product
from pathlib import Path

import numpy as np
import pytest

from helpers import tri_rule_bary, monomial_integral_bary, small_mesh, two_element_mesh

GOLD = Path(__file__).parent / "golden"


def read_gold(name):
    rows = []
    for line in (GOLD / name).read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            rows.append(line.split())
    return rows


def test_basis_orthogonality_and_mass_bruteforce(O):
    """int phi_a phi_b over the reference triangle (area 2) by a 12x12 collapsed Gauss rule:
    diagonal = 2/((2i+1)(i+j+1)) (golden), off-diagonal = 0."""
    lam, wt = tri_rule_bary(12)
    phi = np.array([O.basis(*l)[0] for l in lam])
    M = 2.0 * (phi * wt[:, None]).T @ phi
    gold = [float(r[3]) for r in read_gold("dubiner_closed_forms.txt") if r[0] == "mass"]
    ij = [(0, 0), (0, 1), (1, 0), (0, 2), (1, 1), (2, 0), (0, 3), (1, 2), (2, 1), (3, 0)]
    for k, (i, j) in enumerate(ij):
        assert abs(gold[k] - 2.0 / ((2 * i + 1) * (i + j + 1))) < 1e-15
    assert np.allclose(np.diag(M), gold, rtol=0, atol=1e-14)
    assert np.abs(M - np.diag(np.diag(M))).max() < 1e-14


def test_basis_vertex_values_golden(O):
    rows = [r for r in read_gold("dubiner_closed_forms.txt") if r[0] == "vertex"]
    verts = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
    for r in rows:
        k = int(r[1])
        for v in range(3):
            assert O.basis(*verts[v])[0][k] == float(r[2 + v])
    for p in (1, 2, 3):
        T = O.tables(p)
        pv = T.np("phiV")
        for r in rows:
            k = int(r[1])
            if k < T.ndof:
                assert [pv[v][k] for v in range(3)] == [float(x) for x in r[2:5]]


def test_basis_is_polynomial_of_right_degree_and_derivatives(O):
    """Derivatives d/dxi1, d/dxi2 against central differences; degree of each mode by
    checking that 3rd differences vanish."""
    rng = np.random.default_rng(1)
    for _ in range(20):
        l1, l2 = rng.uniform(0.05, 0.45, 2)
        phi, d1, d2 = O.basis(1 - l1 - l2, l1, l2)
        h = 1e-5   # in lambda; xi = 2 lam - 1 => d/dxi = (1/2) d/dlam
        p1 = O.basis(1 - l1 - h - l2, l1 + h, l2)[0]; m1 = O.basis(1 - l1 + h - l2, l1 - h, l2)[0]
        p2 = O.basis(1 - l1 - l2 - h, l1, l2 + h)[0]; m2 = O.basis(1 - l1 - l2 + h, l1, l2 - h)[0]
        assert np.allclose((p1 - m1) / (2 * h) / 2.0, d1, atol=1e-9)
        assert np.allclose((p2 - m2) / (2 * h) / 2.0, d2, atol=1e-9)
    # modes 0-2 are affine in lambda, modes 3-5 quadratic: exact midpoint identities
    a = np.array([0.2, 0.3, 0.5]); b = np.array([0.6, 0.1, 0.3]); mid = 0.5 * (a + b)
    pa, pb, pm = O.basis(*a)[0], O.basis(*b)[0], O.basis(*mid)[0]
    assert np.allclose(pm[:3], 0.5 * (pa[:3] + pb[:3]), atol=1e-15)
    assert np.abs(pm[3:6] - 0.5 * (pa[3:6] + pb[3:6])).min() > 1e-3      # genuinely quadratic
    # degree along a line: the (n+1)-th finite difference of a degree-n polynomial vanishes, the n-th does not
    ts = np.arange(5) / 4.0
    vals = np.array([O.basis(*(a + t * (b - a)))[0] for t in ts])
    d3 = np.diff(vals, 3, axis=0); d4 = np.diff(vals, 4, axis=0)
    assert np.abs(d3[:, :6]).max() < 1e-13 and np.abs(d4).max() < 1e-13          # modes 0-5: degree <= 2; all: degree <= 3
    assert np.abs(d3[0, 6:]).min() > 1e-3                                             # modes 6-9: genuinely cubic


@pytest.mark.parametrize("p", [1, 2, 3])
def test_area_rule_exact_to_2p_fails_at_2p_plus_1(O, p):
    T = O.tables(p)
    la, wa = T.np("la")[:T.nqa], T.np("wa")[:T.nqa]
    assert abs(wa.sum() - 2.0) < 1e-14
    deg = 2 * p
    for a, b, c in product(range(deg + 2), repeat=3):
        if a + b + c > deg + 1:
            continue
        q = float((wa * la[:, 0] ** a * la[:, 1] ** b * la[:, 2] ** c).sum())
        ex = monomial_integral_bary(a, b, c, area=2.0)
        if a + b + c <= deg:
            assert abs(q - ex) < 2e-14, (a, b, c)
    worst = max(abs(float((wa * la[:, 0] ** a * la[:, 1] ** b * la[:, 2] ** c).sum()) - monomial_integral_bary(a, b, c, 2.0))
                for a, b, c in product(range(deg + 2), repeat=3) if a + b + c == deg + 1)
    assert worst > (1e-4 if p < 3 else 5e-6)      # (the degree-7 monomials' integrals are themselves ~1e-3 at p = 3)


@pytest.mark.parametrize("p", [1, 2, 3])
def test_edge_rule_gauss_legendre_exactness(O, p):
    T = O.tables(p)
    g, w = T.np("ge")[:T.nqe], T.np("we")[:T.nqe]
    assert abs(w.sum() - 2.0) < 1e-15
    for n in range(0, 2 * (p + 1)):
        ex = 0.0 if n % 2 else 2.0 / (n + 1)
        assert abs((w * g ** n).sum() - ex) < 1e-15, n
    n = 2 * (p + 1)
    assert abs((w * g ** n).sum() - 2.0 / (n + 1)) > 1e-3
    el = T.np("elam")[:T.nqe]
    assert np.allclose(el.sum(axis=1), 1.0, atol=1e-16)
    assert np.array_equal(el[:, 0], el[::-1, 1])     # point j of e+ is point nqe-1-j of e-


@pytest.mark.parametrize("p", [1, 2, 3])
def test_tables_are_basis_at_points_and_weights(O, p):
    T = O.tables(p)
    nd = T.ndof
    invM = T.np("invM")[:nd]
    assert np.allclose(1.0 / invM, [2, 1, 1 / 3, 2 / 3, 2 / 9, 2 / 15, 1 / 2, 1 / 6, 1 / 10, 1 / 14][:nd], rtol=1e-15)
    la, wa = T.np("la"), T.np("wa")
    for i in range(T.nqa):
        phi, d1, d2 = O.basis(*la[i])
        assert np.array_equal(T.np("phiA")[i][:nd], phi[:nd])
        assert np.array_equal(T.np("dphiA1")[i][:nd], d1[:nd])
        assert np.array_equal(T.np("dphiA2")[i][:nd], d2[:nd])
        assert np.allclose(T.np("srfac")[i][:nd], wa[i] * invM * phi[:nd], rtol=1e-15)
    el, we = T.np("elam"), T.np("we")
    for l in range(3):
        a, b = (l + 1) % 3, (l + 2) % 3
        for j in range(T.nqe):
            lam = [0.0, 0.0, 0.0]; lam[a] = el[j][0]; lam[b] = el[j][1]
            phi = O.basis(*lam)[0]
            assert np.array_equal(T.np("phiE")[l][j][:nd], phi[:nd])
            assert np.allclose(T.np("efac")[l][j][:nd], we[j] * invM * phi[:nd], rtol=1e-15)


def test_trace_pairing_is_continuous_across_an_edge(O):
    """A globally continuous polynomial field has identical traces from e+ (point j) and
    e- (point nqe-1-j): pins the local-edge / reversed-point convention."""
    from helpers import l2_project
    mesh = small_mesh(nq=3)
    for p in (1, 2):
        T = O.tables(p)
        f = (lambda x, y: 1.0 + 2e-3 * x - 1e-3 * y) if p == 1 else (lambda x, y: 1 + 2e-3 * x - 1e-3 * y + 1e-6 * x * y - 2e-6 * x * x)
        W = l2_project(O, mesh, f, p)
        pe = T.np("phiE")
        for d in range(mesh.n_edge):
            ep, em = mesh.edge_elem[d]
            if em < 0:
                continue
            lp, lm = mesh.edge_local[d]
            for j in range(T.nqe):
                tp = pe[lp][j][:T.ndof] @ W[:, ep]
                tm = pe[lm][T.nqe - 1 - j][:T.ndof] @ W[:, em]
                assert abs(tp - tm) < 1e-9 * max(1.0, abs(tp))


def test_geometry_closure_and_area_sum(O):
    from workloads import c1
    w = c1(nq=8)
    o = O.Oracle.from_workload(w)
    area, jinv, lfac, enx, eny = o.get_geometry()
    assert abs(area.sum() - 1.0e8) < 1e-4
    mesh = small_mesh(nq=4)
    o = O.Oracle(dict(p=1, rk_order=2, g=9.81, cf=0, coriolis_f=0, h0_dry=1e-3, limiter=0, wetdry=0),
                 mesh.xy, np.full(mesh.n_nodes, 10.0), mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)
    area, jinv, lfac, enx, eny = o.get_geometry()
    assert abs(area.sum() - 1.0e6) < 1e-6
    assert np.allclose(np.hypot(enx, eny), 1.0, atol=1e-15)
    for e in range(mesh.n_elem):
        s = np.zeros(2)
        for l in range(3):
            d = mesh.elem_edge[e, l]
            sign = 1.0 if (mesh.edge_elem[d, 0] == e and mesh.edge_local[d, 0] == l) else -1.0
            s += sign * lfac[l, e] * area[e] * np.array([enx[d], eny[d]])      # L_l n_l
        assert np.abs(s).max() < 1e-9
        # jinv rows are grad xi_1, grad xi_2: check against finite geometry
        X = mesh.xy[mesh.tri[e]]
        J = 0.5 * np.array([[X[1][0] - X[0][0], X[2][0] - X[0][0]], [X[1][1] - X[0][1], X[2][1] - X[0][1]]])
        Ji = np.linalg.inv(J)
        assert np.allclose([[jinv[0, e], jinv[1, e]], [jinv[2, e], jinv[3, e]]], Ji, rtol=1e-12)


def test_paper_structural_facts(O):
    facts = {r[0]: float(r[1]) for r in read_gold("paper_facts.txt")}
    T = O.tables(1)
    assert 3 * T.ndof == facts["dofs_per_element_p1"]
    assert facts["harvey_elements"] * facts["dofs_per_element_p1"] == 60079653
    m = two_element_mesh()
    assert m.elem_edge.shape[1] == facts["local_edges_per_element"]
    inter = m.edge_elem[:, 1] >= 0
    assert inter.sum() == 1 and set(m.edge_local[inter].ravel()) <= {0, 1, 2}
