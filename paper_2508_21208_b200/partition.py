"""Domain decomposition of a triangular mesh for the DG-SWEM stage (host side, numpy; DESIGN.md section 10;
PAPER.md:476-519 "Multiple GPUs": one subdomain per GPU, ghost elements refreshed every RK stage).

`partition(mesh tables, n_parts)` cuts the elements into `n_parts` contiguous chunks of a space-filling (Morton) order of
their centroids and returns, for every part, a self-contained local mesh in the form `dgswem_create` takes:

  * local elements = the part's OWNED elements (in ascending global id) followed by its GHOST elements: the
    edge-neighbours of owned elements that belong to other parts (one layer: all the stage needs of a neighbour is its
    state, and all the edge-neighbour limiter needs is its mean) -- or, with ghost="vertex", every foreign element that
    shares a NODE with an owned element: the vertex-neighbourhood limiter (limiter = 2, R-18) bounds an
    element by the means of all elements around its three vertices;
  * an edge with both elements local keeps its global orientation (e+, e-); an edge whose other element is not local --
    the outer edges of ghost elements -- is closed as a land edge of the local element (its result is never used: ghost
    elements are overwritten by every exchange); true boundary edges keep their code;
  * `send[q]` / `recv[q]`: local ids of the owned elements part q holds as ghosts / of the ghosts owned by part q, both in
    ascending global id, so that the k-th value sent is the k-th value expected.

No arithmetic of the method lives here; this is index bookkeeping only.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class SubMesh:
    part: int
    xy: np.ndarray            # [n_nodes_local, 2]
    node_gid: np.ndarray      # [n_nodes_local] global node ids
    tri: np.ndarray           # [n_local, 3] local node ids, vertex order as in the global mesh
    edge_elem: np.ndarray     # [n_edge_local, 2]
    edge_local: np.ndarray    # [n_edge_local, 2] int8
    edge_bc: np.ndarray       # [n_edge_local]
    elem_edge: np.ndarray     # [n_local, 3]
    elem_gid: np.ndarray      # [n_local] global element ids: owned first, then ghosts
    n_owned: int
    send: dict = field(default_factory=dict)   # q -> local ids (owned) to pack for part q
    recv: dict = field(default_factory=dict)   # q -> local ids (ghosts) to unpack from part q

    @property
    def n_local(self) -> int:
        return int(self.elem_gid.size)

    def halo_lists(self):
        """Concatenated send / receive lists in ascending peer order, and the per-peer counts."""
        peers = sorted(set(self.send) | set(self.recv))
        snd = np.concatenate([self.send.get(q, np.empty(0, np.int32)) for q in peers]) if peers else np.empty(0, np.int32)
        rcv = np.concatenate([self.recv.get(q, np.empty(0, np.int32)) for q in peers]) if peers else np.empty(0, np.int32)
        return (snd.astype(np.int32), rcv.astype(np.int32), peers,
                [int(self.send.get(q, np.empty(0)).size) for q in peers], [int(self.recv.get(q, np.empty(0)).size) for q in peers])


def _morton_order(cx: np.ndarray, cy: np.ndarray) -> np.ndarray:
    def spread(v):
        v = v.astype(np.uint64)
        v = (v | (v << np.uint64(16))) & np.uint64(0x0000FFFF0000FFFF)
        v = (v | (v << np.uint64(8))) & np.uint64(0x00FF00FF00FF00FF)
        v = (v | (v << np.uint64(4))) & np.uint64(0x0F0F0F0F0F0F0F0F)
        v = (v | (v << np.uint64(2))) & np.uint64(0x3333333333333333)
        v = (v | (v << np.uint64(1))) & np.uint64(0x5555555555555555)
        return v
    span = max(cx.max() - cx.min(), cy.max() - cy.min(), 1e-300)
    ix = np.minimum(65535, ((cx - cx.min()) / span * 65535.0)).astype(np.uint64)
    iy = np.minimum(65535, ((cy - cy.min()) / span * 65535.0)).astype(np.uint64)
    return np.argsort(spread(ix) | (spread(iy) << np.uint64(1)), kind="stable")


def element_parts(xy, tri, n_parts: int) -> np.ndarray:
    """part id of every element: equal-size contiguous chunks of the Morton order of the centroids."""
    c = xy[tri].mean(axis=1)
    order = _morton_order(c[:, 0], c[:, 1])
    part = np.empty(tri.shape[0], dtype=np.int32)
    bounds = np.linspace(0, tri.shape[0], n_parts + 1).astype(np.int64)
    for p in range(n_parts):
        part[order[bounds[p]:bounds[p + 1]]] = p
    return part


def partition(xy, tri, edge_elem, edge_local, edge_bc, elem_edge, n_parts: int, part: np.ndarray | None = None,
              ghost: str = "edge"):
    """Split the mesh into `n_parts` SubMesh objects (see the module docstring).  `part` overrides the element -> part map;
    ghost = "edge" (edge-neighbours of owned elements) or "vertex" (every foreign element around a node of an owned one)."""
    if ghost not in ("edge", "vertex"):
        raise ValueError("ghost must be 'edge' or 'vertex'")
    xy = np.asarray(xy, dtype=np.float64)
    tri = np.asarray(tri, dtype=np.int32)
    edge_elem = np.asarray(edge_elem, dtype=np.int32)
    edge_local = np.asarray(edge_local, dtype=np.int8)
    edge_bc = np.asarray(edge_bc, dtype=np.int32)
    elem_edge = np.asarray(elem_edge, dtype=np.int32)
    ne = tri.shape[0]
    if part is None:
        part = element_parts(xy, tri, n_parts)
    part = np.asarray(part, dtype=np.int32)
    if part.shape != (ne,) or part.min() < 0 or part.max() >= n_parts:
        raise ValueError("part must assign every element to a part in [0, n_parts)")
    ep, em = edge_elem[:, 0].astype(np.int64), edge_elem[:, 1].astype(np.int64)
    interior = em >= 0
    part_p = part[ep]
    part_m = np.where(interior, part[np.maximum(em, 0)], -1)
    subs, g2l_all = [], []
    for p in range(n_parts):
        owned = np.flatnonzero(part == p)
        if owned.size == 0:
            raise ValueError(f"part {p} owns no element")
        in_p, in_m = part_p == p, part_m == p
        cut = interior & (in_p != in_m)
        ghosts = np.unique(np.where(in_p[cut], em[cut], ep[cut]))
        if ghost == "vertex":
            touched = np.zeros(xy.shape[0], dtype=bool)
            touched[tri[owned].ravel()] = True
            ghosts = np.flatnonzero(touched[tri].any(axis=1) & (part != p))      # ascending global id; contains the edge-neighbours
        elem_gid = np.concatenate([owned, ghosts]).astype(np.int64)
        g2l = np.full(ne, -1, dtype=np.int64)
        g2l[elem_gid] = np.arange(elem_gid.size)
        ed = np.unique(elem_edge[elem_gid].ravel()).astype(np.int64)
        eg2l = np.full(edge_elem.shape[0], -1, dtype=np.int64)
        eg2l[ed] = np.arange(ed.size)
        lep = g2l[ep[ed]]
        lem = np.where(em[ed] >= 0, g2l[np.maximum(em[ed], 0)], -1)
        only_m = (lep < 0) & (lem >= 0)           # only the global e- side is local: it becomes the e+ of a closed edge
        both = (lep >= 0) & (lem >= 0)
        ee = np.stack([np.where(only_m, lem, lep), np.where(both, lem, -1)], axis=1).astype(np.int32)
        el = np.stack([np.where(only_m, edge_local[ed, 1], edge_local[ed, 0]),
                       np.where(both, edge_local[ed, 1], -1)], axis=1).astype(np.int8)
        true_boundary = em[ed] < 0
        bc = np.where(both, 0, np.where(true_boundary, edge_bc[ed], 1)).astype(np.int32)
        node_gid = np.unique(tri[elem_gid].ravel())
        tri_l = np.searchsorted(node_gid, tri[elem_gid]).astype(np.int32)
        subs.append(SubMesh(part=p, xy=xy[node_gid].copy(), node_gid=node_gid, tri=tri_l, edge_elem=ee, edge_local=el,
                            edge_bc=bc, elem_edge=eg2l[elem_edge[elem_gid]].astype(np.int32), elem_gid=elem_gid,
                            n_owned=int(owned.size)))
        g2l_all.append(g2l)
    for p, sm in enumerate(subs):
        ghosts = sm.elem_gid[sm.n_owned:]
        owner = part[ghosts]
        for q in np.unique(owner):
            gids = ghosts[owner == q]                                   # ascending global id
            sm.recv[int(q)] = g2l_all[p][gids].astype(np.int32)
            subs[int(q)].send[p] = g2l_all[int(q)][gids].astype(np.int32)
    return subs
