"""Seeded synthetic triangulations and the precomputed edge/neighbour tables.

This module serves BOTH the CPU oracle and the CUDA path (it is the "seeded
input generator" module): it produces node coordinates, triangle connectivity
and the edge tables that `dgswem_create` takes (the tables are
the paper's NEDEL / LED / NIEDN, Alg. 2 lines 4-9).  It holds
none of the method's arithmetic (no basis, quadrature, flux or time stepping).

Conventions:
  * triangles are counter-clockwise, 0-based node ids;
  * local edge l of an element joins local vertices (l+1)%3 -> (l+2)%3
    (it is opposite local vertex l);
  * edge_elem[d] = (e+, e-), e- = -1 on a boundary edge;
    edge_local[d] = (local edge of e+, local edge of e- or -1);
    edge_bc[d] = 0 interior, 1 land/wall, 2 ocean elevation;
    elem_edge[e][l] = global edge of local edge l.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Mesh:
    xy: np.ndarray          # [n_nodes, 2] float64
    tri: np.ndarray         # [n_elem, 3] int32, CCW
    edge_elem: np.ndarray   # [n_edge, 2] int32
    edge_local: np.ndarray  # [n_edge, 2] int8
    edge_bc: np.ndarray     # [n_edge] int32
    elem_edge: np.ndarray   # [n_elem, 3] int32
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return int(self.xy.shape[0])

    @property
    def n_elem(self) -> int:
        return int(self.tri.shape[0])

    @property
    def n_edge(self) -> int:
        return int(self.edge_elem.shape[0])


def signed_areas(xy: np.ndarray, tri: np.ndarray) -> np.ndarray:
    """Signed triangle areas (generator-side validity check only)."""
    p0, p1, p2 = xy[tri[:, 0]], xy[tri[:, 1]], xy[tri[:, 2]]
    return 0.5 * ((p1[:, 0] - p0[:, 0]) * (p2[:, 1] - p0[:, 1])
                  - (p2[:, 0] - p0[:, 0]) * (p1[:, 1] - p0[:, 1]))


def grid_nodes(nx_nodes: int, ny_nodes: int, lx: float, ly: float,
               x_coords: np.ndarray | None = None) -> np.ndarray:
    """Node coordinates of an nx_nodes x ny_nodes grid, node id = j*nx_nodes + i."""
    xs = np.linspace(0.0, lx, nx_nodes) if x_coords is None else np.asarray(x_coords, dtype=np.float64)
    ys = np.linspace(0.0, ly, ny_nodes)
    X, Y = np.meshgrid(xs, ys, indexing="xy")
    return np.stack([X.ravel(), Y.ravel()], axis=1).astype(np.float64)


def jitter_interior(xy: np.ndarray, nx_nodes: int, ny_nodes: int, frac: float,
                    rng: np.random.Generator) -> np.ndarray:
    """Move interior nodes by U(-frac, frac) x local cell size; boundary nodes stay put."""
    xy = xy.copy().reshape(ny_nodes, nx_nodes, 2)
    # local cell size per node = mean of the spacing to the two grid neighbours
    dx = np.zeros((ny_nodes, nx_nodes))
    dy = np.zeros((ny_nodes, nx_nodes))
    dx[:, 1:-1] = np.minimum(xy[:, 2:, 0] - xy[:, 1:-1, 0], xy[:, 1:-1, 0] - xy[:, :-2, 0])
    dy[1:-1, :] = np.minimum(xy[2:, :, 1] - xy[1:-1, :, 1], xy[1:-1, :, 1] - xy[:-2, :, 1])
    jx = rng.uniform(-frac, frac, size=(ny_nodes, nx_nodes)) * dx
    jy = rng.uniform(-frac, frac, size=(ny_nodes, nx_nodes)) * dy
    jx[0, :] = jx[-1, :] = 0.0
    jx[:, 0] = jx[:, -1] = 0.0
    jy[0, :] = jy[-1, :] = 0.0
    jy[:, 0] = jy[:, -1] = 0.0
    xy[:, :, 0] += jx
    xy[:, :, 1] += jy
    return xy.reshape(-1, 2)


def split_quads(nx_nodes: int, ny_nodes: int, diag: np.ndarray | int) -> np.ndarray:
    """Split every grid quad into two CCW triangles.

    diag: 0 -> all quads cut along n00-n11; 1 -> all along n10-n01; or an
    int array [(ny_nodes-1)*(nx_nodes-1)] of 0/1 per quad (row-major in j, i).
    Elements 2q and 2q+1 belong to quad q.
    """
    nqx, nqy = nx_nodes - 1, ny_nodes - 1
    i, j = np.meshgrid(np.arange(nqx), np.arange(nqy), indexing="xy")
    i, j = i.ravel(), j.ravel()
    n00 = j * nx_nodes + i
    n10 = n00 + 1
    n01 = n00 + nx_nodes
    n11 = n01 + 1
    d = np.broadcast_to(np.asarray(diag), n00.shape).astype(bool)
    ta = np.where(d[:, None], np.stack([n00, n10, n01], 1), np.stack([n00, n10, n11], 1))
    tb = np.where(d[:, None], np.stack([n10, n11, n01], 1), np.stack([n00, n11, n01], 1))
    tri = np.empty((2 * n00.size, 3), dtype=np.int32)
    tri[0::2] = ta
    tri[1::2] = tb
    return tri


def build_edge_tables(tri: np.ndarray, n_nodes: int):
    """edge_elem, edge_local, elem_edge from connectivity (all boundary edges get bc=1).

    e+ of an interior edge is the side with the smaller element id; edges are
    numbered in ascending (min node, max node) order.
    """
    n_elem = tri.shape[0]
    tri64 = tri.astype(np.int64)
    a = np.stack([tri64[:, 1], tri64[:, 2], tri64[:, 0]], axis=1)  # local edge l: (l+1)%3
    b = np.stack([tri64[:, 2], tri64[:, 0], tri64[:, 1]], axis=1)  #               (l+2)%3
    lo = np.minimum(a, b).ravel()
    hi = np.maximum(a, b).ravel()
    key = lo * np.int64(n_nodes) + hi
    elem = np.repeat(np.arange(n_elem, dtype=np.int64), 3)
    loc = np.tile(np.arange(3, dtype=np.int64), n_elem)
    order = np.lexsort((elem, key))
    key_s, elem_s, loc_s = key[order], elem[order], loc[order]
    first = np.ones(key_s.size, dtype=bool)
    first[1:] = key_s[1:] != key_s[:-1]
    edge_id_s = np.cumsum(first) - 1
    n_edge = int(edge_id_s[-1]) + 1
    counts = np.bincount(edge_id_s, minlength=n_edge)
    if counts.max() > 2:
        raise ValueError("non-manifold mesh: an edge has more than two elements")
    edge_elem = np.full((n_edge, 2), -1, dtype=np.int32)
    edge_local = np.full((n_edge, 2), -1, dtype=np.int8)
    side = (~first).astype(np.int64)  # 0 for the first (smaller element id), 1 for the second
    edge_elem[edge_id_s, side] = elem_s
    edge_local[edge_id_s, side] = loc_s
    elem_edge = np.empty((n_elem, 3), dtype=np.int32)
    elem_edge[elem_s, loc_s] = edge_id_s
    edge_bc = np.where(edge_elem[:, 1] < 0, 1, 0).astype(np.int32)
    return edge_elem, edge_local, edge_bc, elem_edge


def permute_elements(tri: np.ndarray, rng: np.random.Generator) -> tuple[np.ndarray, np.ndarray]:
    """Random element renumbering (mimics unstructured indexing). Returns (tri_new, perm)
    with tri_new[i] = tri[perm[i]]."""
    perm = rng.permutation(tri.shape[0])
    return np.ascontiguousarray(tri[perm]), perm


def permute_edges(edge_elem, edge_local, edge_bc, elem_edge, rng: np.random.Generator):
    """Random renumbering of the global edges (keeps all tables consistent)."""
    n_edge = edge_elem.shape[0]
    perm = rng.permutation(n_edge)          # new edge i = old edge perm[i]
    inv = np.empty(n_edge, dtype=np.int64)
    inv[perm] = np.arange(n_edge)
    return (np.ascontiguousarray(edge_elem[perm]), np.ascontiguousarray(edge_local[perm]),
            np.ascontiguousarray(edge_bc[perm]), inv[elem_edge].astype(np.int32))


def make_mesh(xy: np.ndarray, tri: np.ndarray, *, ocean_pred=None, shuffle_edges_rng=None,
              meta: dict | None = None) -> Mesh:
    """Assemble a Mesh: edge tables, boundary codes (ocean where ocean_pred(xm, ym) is true)."""
    areas = signed_areas(xy, tri)
    if not (areas > 0).all():
        raise ValueError("generator produced a non-CCW or degenerate triangle")
    edge_elem, edge_local, edge_bc, elem_edge = build_edge_tables(tri, xy.shape[0])
    if ocean_pred is not None:
        bnd = np.nonzero(edge_elem[:, 1] < 0)[0]
        ep = edge_elem[bnd, 0]
        lp = edge_local[bnd, 0].astype(np.int64)
        na = tri[ep, (lp + 1) % 3]
        nb = tri[ep, (lp + 2) % 3]
        xm = 0.5 * (xy[na, 0] + xy[nb, 0])
        ym = 0.5 * (xy[na, 1] + xy[nb, 1])
        edge_bc[bnd[ocean_pred(xm, ym)]] = 2
    if shuffle_edges_rng is not None:
        edge_elem, edge_local, edge_bc, elem_edge = permute_edges(
            edge_elem, edge_local, edge_bc, elem_edge, shuffle_edges_rng)
    return Mesh(np.ascontiguousarray(xy, dtype=np.float64), np.ascontiguousarray(tri, dtype=np.int32),
                edge_elem, edge_local, edge_bc, elem_edge, dict(meta or {}))


def rect_mesh(nqx: int, nqy: int, lx: float, ly: float, *, diag="same", jitter=0.0,
              permute=False, rng: np.random.Generator | None = None, ocean_pred=None,
              x_coords=None, meta=None) -> Mesh:
    """nqx x nqy quads on [0,lx]x[0,ly], each split into two triangles.

    diag: "same" (all n00-n11), "random" (Bernoulli 1/2 per quad, seeded).
    jitter: interior nodes moved by U(-jitter, jitter) x local cell size.
    permute: random element and edge renumbering (seeded).
    """
    nxn, nyn = nqx + 1, nqy + 1
    xy = grid_nodes(nxn, nyn, lx, ly, x_coords)
    if diag == "random":
        assert rng is not None
        d = rng.integers(0, 2, size=nqx * nqy)
    elif diag == "same":
        d = 0
    else:
        raise ValueError(diag)
    if jitter > 0.0:
        assert rng is not None
        xy = jitter_interior(xy, nxn, nyn, jitter, rng)
    tri = split_quads(nxn, nyn, d)
    if jitter > 0.0:
        # A jittered quad can be non-convex or nearly so: where the drawn diagonal gives a
        # triangle smaller than 15 % of the mean of the quad's two triangles, take the
        # other diagonal if its smaller triangle is larger.
        alt = split_quads(nxn, nyn, 1 - np.broadcast_to(np.asarray(d), (nqx * nqy,)))
        a0 = signed_areas(xy, tri).reshape(-1, 2)
        a1 = signed_areas(xy, alt).reshape(-1, 2)
        bad = a0.min(axis=1) < 0.15 * a0.mean(axis=1)
        flip = bad & (a1.min(axis=1) > a0.min(axis=1))
        tri = np.where(np.repeat(flip, 2)[:, None], alt, tri).astype(np.int32)
    if permute:
        assert rng is not None
        tri, _ = permute_elements(tri, rng)
    return make_mesh(xy, tri, ocean_pred=ocean_pred,
                     shuffle_edges_rng=rng if permute else None, meta=meta)


def vertex_to_modal_p1(u_nodes: np.ndarray, tri: np.ndarray, ndof: int) -> np.ndarray:
    """Modal coefficients [ndof, n_elem] of the element-wise linear interpolant of a
    nodal field (input preparation only).  With vertex values (u0,u1,u2) the linear
    Dubiner modes (order 00, 01, 10) are a=(u0+u1+u2)/3,
    b=(u2-a)/2, c=(u1-u0)/2; higher modes are zero."""
    u0, u1, u2 = u_nodes[tri[:, 0]], u_nodes[tri[:, 1]], u_nodes[tri[:, 2]]
    out = np.zeros((ndof, tri.shape[0]), dtype=np.float64)
    a = (u0 + u1 + u2) / 3.0
    out[0] = a
    out[1] = 0.5 * (u2 - a)
    out[2] = 0.5 * (u1 - u0)
    return out
