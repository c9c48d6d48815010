"""Pins for the vertex-neighbourhood (linearity-preserving) slope limiter, prm.limiter = 2 (SURVEY.md 8(c.2) "known
weakness", 8(f) NEXT-3; "optional slope limiter"; R-18).  Expected values are recomputed in numpy
from the mesh's node lists; the defining property -- a linear field is left untouched away from the boundary, which
the edge-neighbour limiter of R-7 does not achieve on a jittered mesh -- is checked bit for bit."""
import numpy as np
import pytest

from helpers import small_mesh
from workloads import c4, default_params
from workloads.configs import _modal


def make_oracle(O, mesh, bathy, **kw):
    prm = default_params(**kw)
    return O.Oracle(prm, mesh.xy, bathy, mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)


def _np_alpha(w3, lo, hi):
    a, b, c = w3
    alpha = 1.0
    for v, d in enumerate((-b - c, -b + c, 2 * b)):
        if d > 0:
            alpha = min(alpha, (hi[v] - a) / d)
        elif d < 0:
            alpha = min(alpha, (lo[v] - a) / d)
    return alpha


def test_limit_var_vertex_properties(O):
    rng = np.random.default_rng(0)
    phiV = np.array([[1, -1, -1], [1, -1, 1], [1, 2, 0]], dtype=float)
    n_active = 0
    for _ in range(400):
        w = rng.normal(size=3) * [1.0, 0.5, 0.5]
        lo = w[0] - np.abs(rng.normal(size=3)) * 0.4
        hi = w[0] + np.abs(rng.normal(size=3)) * 0.4
        alpha, wl = O.limit_var_vertex(1, w, lo, hi)
        assert 0.0 <= alpha <= 1.0 and wl[0] == w[0]
        assert abs(alpha - _np_alpha(w, lo, hi)) <= 1e-15
        v = phiV @ wl
        assert (v <= hi + 1e-14).all() and (v >= lo - 1e-14).all()      # each vertex inside ITS OWN bounds
        v0 = phiV @ w
        if (v0 <= hi).all() and (v0 >= lo).all():
            assert alpha == 1.0 and np.array_equal(wl, w)
        else:
            n_active += 1
            assert alpha < 1.0
    assert n_active > 100
    a, wl = O.limit_var_vertex(2, [1.0, 2.0, 0.0, 0.3, 0.2, 0.1], [0.9] * 3, [1.1] * 3)
    assert a < 1 and np.array_equal(wl[3:], [0, 0, 0])
    a, wl = O.limit_var_vertex(2, [1.0, 1e-3, 0.0, 0.3, 0.2, 0.1], [0.9] * 3, [1.1] * 3)
    assert a == 1 and np.array_equal(wl[3:], [0.3, 0.2, 0.1])


def _node_extrema(mesh, means):
    lo = np.full(mesh.n_nodes, np.inf); hi = np.full(mesh.n_nodes, -np.inf)
    np.minimum.at(lo, mesh.tri.ravel(), np.repeat(means, 3))
    np.maximum.at(hi, mesh.tri.ravel(), np.repeat(means, 3))
    return lo, hi


@pytest.mark.parametrize("p", [1, 2])
def test_vertex_limiter_wiring_through_the_model(O, p):
    """limiter_all with limiter = 2 on a jittered, permuted 32-element mesh: alpha of every (element, variable) from
    numpy node extrema (np.minimum.at over mesh.tri); a dry-flagged element is skipped but its mean still counts in the
    extrema of its nodes; means never change."""
    mesh = small_mesh(nq=4, L=2000.0, seed=31)
    rng = np.random.default_rng(31)
    nd = (p + 1) * (p + 2) // 2
    st = np.zeros((3, nd, mesh.n_elem))
    st[:, 0] = rng.uniform(-1, 1, (3, mesh.n_elem))
    st[:, 1:3] = 0.4 * rng.uniform(-1, 1, (3, 2, mesh.n_elem))
    if p == 2:
        st[:, 3:] = 0.05 * rng.uniform(-1, 1, (3, 3, mesh.n_elem))
    o = make_oracle(O, mesh, np.full(mesh.n_nodes, 20.0), p=p, limiter=2, wetdry=1)
    wet = np.ones(mesh.n_elem, dtype=np.uint8)
    dry_e = 9
    st[0, 0, dry_e] = 5.0                                       # an extreme mean in the dry element: it must still bound its neighbours
    wet[dry_e] = 0
    o.set_state_raw(0.0, *st, wet)
    o.apply_post(limiter=True, wetdry=False)
    _, *out = o.get_state()
    out = np.stack(out)
    assert np.array_equal(out[:, 0], st[:, 0])
    assert np.array_equal(out[:, :, dry_e], st[:, :, dry_e])
    n_bind = 0
    for c in range(3):
        lo, hi = _node_extrema(mesh, st[c, 0])
        for e in range(mesh.n_elem):
            if e == dry_e:
                continue
            nodes = mesh.tri[e]
            alpha = _np_alpha(st[c, :3, e], lo[nodes], hi[nodes])
            n_bind += alpha < 1.0
            assert np.abs(out[c, 1:3, e] - alpha * st[c, 1:3, e]).max() <= 1e-15
            if p == 2:
                assert np.array_equal(out[c, 3:, e], np.zeros(3) if alpha < 1.0 else st[c, 3:, e])
    assert n_bind > 20
    # the dry element's mean (5.0) is the upper bound at its three nodes
    lo, hi = _node_extrema(mesh, st[0, 0])
    assert (hi[mesh.tri[dry_e]] == 5.0).all()


def test_linear_field_is_preserved_where_the_edge_neighbour_limiter_fails(O):
    """Linearity preservation (the property SURVEY 8(c.2) says the edge-neighbour Barth-Jespersen lacks on general
    meshes): a globally linear field on a jittered mesh is left bit-for-bit unchanged by limiter = 2 in every element
    without a boundary node (each interior vertex lies in the convex hull of the centroids around it), while
    limiter = 1 clips some of those same elements."""
    mesh = small_mesh(nq=10, L=5000.0, jitter=0.3, seed=77)
    f = [lambda x, y: 0.2 + 3e-4 * x - 2e-4 * y, lambda x, y: 1.0 - 4e-4 * x + 1e-4 * y, lambda x, y: -0.5 + 2e-4 * x + 5e-4 * y]
    st = [_modal(fi(mesh.xy[:, 0], mesh.xy[:, 1]), mesh, 1) for fi in f]
    bnd_node = np.zeros(mesh.n_nodes, dtype=bool)
    for d in np.flatnonzero(mesh.edge_bc != 0):
        e, l = mesh.edge_elem[d, 0], mesh.edge_local[d, 0]
        bnd_node[mesh.tri[e, (l + 1) % 3]] = True; bnd_node[mesh.tri[e, (l + 2) % 3]] = True
    interior = ~bnd_node[mesh.tri].any(axis=1)
    assert interior.sum() > 80
    wet = np.ones(mesh.n_elem, dtype=np.uint8)
    changed = {}
    for lim in (1, 2):
        o = make_oracle(O, mesh, np.full(mesh.n_nodes, 30.0), p=1, limiter=lim)
        o.set_state_raw(0.0, *st, wet)
        o.apply_post(limiter=True, wetdry=False)
        _, *out = o.get_state()
        changed[lim] = np.array([(np.stack(out)[:, :, e] != np.stack(st)[:, :, e]).any() for e in range(mesh.n_elem)])
    assert not changed[2][interior].any()                     # linearity preserved, bit for bit
    assert changed[1][interior].sum() >= 3                    # the edge-neighbour limiter clips a linear field


def test_vertex_limiter_in_a_run_conserves_mass(O):
    w = c4(nqx=32, nqy=16, nsteps=40)
    prm = dict(w.params); prm["limiter"] = 2
    m = w.mesh
    o = O.Oracle(prm, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    o.set_wind_holland(w.holland)
    o.set_state(0.0, w.ze, w.qx, w.qy)
    area = o.get_geometry()[0]
    _, z, _, _ = o.get_state()
    m0 = float((area * z[0]).sum())
    vol = float((area * np.maximum(z[0] + w.bathy[m.tri].mean(axis=1), 0)).sum())
    o.step(40, w.dt)
    _, z, qx, qy = o.get_state()
    assert np.isfinite(z).all() and np.abs(qx).max() > 1e-6
    assert abs(float((area * z[0]).sum()) - m0) < 1e-12 * vol
    o1 = O.Oracle.from_workload(w); o1.step(40, w.dt)
    assert np.abs(o1.get_state()[2] - qx).max() > 1e-9          # a different limiter gives a different run
