"""Host-side domain decomposition (paper_2508_21208_b200/partition.py, decomp.py transports): invariants of the
partitions and halo plans, the library's own mesh validation of every local mesh, and the multi-rank transport on CPU
(gloo, world_size 2 and 3)."""
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _mesh():
    from workloads import c3
    return c3(nn=30)


@pytest.mark.parametrize("n_parts", [2, 3, 7])
def test_partition_invariants(n_parts):
    from paper_2508_21208_b200.partition import partition
    w = _mesh(); m = w.mesh
    subs = partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, n_parts)
    owned = np.concatenate([s.elem_gid[:s.n_owned] for s in subs])
    assert np.array_equal(np.sort(owned), np.arange(m.n_elem))             # every element owned exactly once
    nbr = {}                                                                # edge-neighbours of every element
    for (a, b) in m.edge_elem:
        if b >= 0:
            nbr.setdefault(int(a), set()).add(int(b)); nbr.setdefault(int(b), set()).add(int(a))
    for s in subs:
        own = set(s.elem_gid[:s.n_owned].tolist())
        ghosts = set(s.elem_gid[s.n_owned:].tolist())
        want = set().union(*[nbr.get(e, set()) for e in own]) - own
        assert ghosts == want                                               # exactly one layer of edge-neighbours
        assert np.array_equal(m.tri[s.elem_gid], s.node_gid[s.tri])         # same triangles, same vertex order
        # local tables are mutually consistent and every owned element's edges keep their global meaning
        for le in range(s.n_local):
            for l in range(3):
                d = s.elem_edge[le, l]
                side = 0 if (s.edge_elem[d, 0] == le and s.edge_local[d, 0] == l) else 1
                assert s.edge_elem[d, side] == le and s.edge_local[d, side] == l
                gd = m.elem_edge[s.elem_gid[le], l]
                if le < s.n_owned:
                    ge = m.edge_elem[gd]
                    if ge[1] >= 0:                                          # interior globally: both sides local, same orientation
                        assert np.array_equal(s.elem_gid[s.edge_elem[d]], ge) and s.edge_bc[d] == 0
                    else:
                        assert s.edge_elem[d, 1] == -1 and s.edge_bc[d] == m.edge_bc[gd]
        # halo lists: what q sends to p is what p expects from q, element by element
        for q, ids in s.recv.items():
            assert np.array_equal(s.elem_gid[ids], subs[q].elem_gid[subs[q].send[s.part]])
            assert (ids >= s.n_owned).all() and (subs[q].send[s.part] < subs[q].n_owned).all()
        assert sum(v.size for v in s.recv.values()) == s.n_local - s.n_owned


@pytest.mark.parametrize("n_parts", [2, 5])
def test_vertex_ghost_layer_for_the_vertex_limiter(n_parts):
    """ghost="vertex" (what PartitionedDgswem uses with limiter = 2): the ghosts of a part are exactly the foreign elements
    that share a node with one of its owned elements -- so every node of an owned element has, locally, the same set of
    incident elements as in the whole mesh (what the node extrema of DESIGN.md R-18 are taken over) -- the
    edge-neighbour layer is contained in it, and the halo lists still pair up element by element."""
    from paper_2508_21208_b200.partition import partition
    w = _mesh(); m = w.mesh
    edge_subs = partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, n_parts)
    subs = partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, n_parts, ghost="vertex")
    around = [set() for _ in range(m.n_nodes)]
    for e, t in enumerate(m.tri):
        for n in t:
            around[n].add(e)
    for s, se in zip(subs, edge_subs):
        own = set(s.elem_gid[:s.n_owned].tolist())
        ghosts = set(s.elem_gid[s.n_owned:].tolist())
        want = set().union(*[around[n] for e in own for n in m.tri[e]]) - own
        assert ghosts == want and ghosts >= set(se.elem_gid[se.n_owned:].tolist()) and len(ghosts) > se.n_local - se.n_owned
        local = set(s.elem_gid.tolist())
        for e in own:
            for n in m.tri[e]:
                assert around[n] <= local
        assert np.array_equal(m.tri[s.elem_gid], s.node_gid[s.tri])
        for q, ids in s.recv.items():
            assert np.array_equal(s.elem_gid[ids], subs[q].elem_gid[subs[q].send[s.part]])
            assert (ids >= s.n_owned).all() and (subs[q].send[s.part] < subs[q].n_owned).all()
        assert sum(v.size for v in s.recv.values()) == s.n_local - s.n_owned
    with pytest.raises(ValueError):
        partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, 2, ghost="node")


def test_local_meshes_pass_the_library_validation():
    """dgswem_create validates tables on the host before touching CUDA: every local mesh must get past it."""
    import ctypes as C
    import torch
    from paper_2508_21208_b200 import build, load_library
    from paper_2508_21208_b200.binding import Params
    from paper_2508_21208_b200.partition import partition
    build.build()
    lib = load_library()
    w = _mesh(); m = w.mesh
    prm = w.params
    P = Params(p=int(prm["p"]), rk_order=int(prm["rk_order"]), g=prm["g"], cf=prm["cf"], coriolis_f=prm["coriolis_f"],
               h0_dry=prm["h0_dry"], limiter=int(prm["limiter"]), wetdry=int(prm["wetdry"]), reorder=1, device=0)
    for s in partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, 4):
        xy = np.ascontiguousarray(s.xy); b = np.ascontiguousarray(w.bathy[s.node_gid])
        tri = np.ascontiguousarray(s.tri); ee = np.ascontiguousarray(s.edge_elem); el = np.ascontiguousarray(s.edge_local)
        bc = np.ascontiguousarray(s.edge_bc); eled = np.ascontiguousarray(s.elem_edge)
        dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double)); ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        h = C.c_void_p()
        rc = lib.dgswem_create(C.byref(h), C.byref(P), None, xy.shape[0], dp(xy), dp(b), tri.shape[0], ip(tri), ee.shape[0], ip(ee),
                               el.ctypes.data_as(C.POINTER(C.c_int8)), ip(bc), ip(eled))
        assert rc == (0 if torch.cuda.is_available() else -3), lib.dgswem_last_error(None)
        if rc == 0:
            lib.dgswem_destroy(h)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from paper_2508_21208_b200.partition import partition
    from paper_2508_21208_b200.decomp import HaloPlan, DistTransport
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        w = _mesh(); m = w.mesh
        sub = partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, world)[rank]
        plan = HaloPlan(sub)
        rows = 3
        # every rank "packs" a code of the global id of each element it sends: row r carries gid * 10 + r
        gid_s = torch.from_numpy(sub.elem_gid[plan.send_ids].astype(np.float64))
        snd = torch.stack([gid_s * 10 + r for r in range(rows)])
        rcv = torch.full((rows, plan.n_recv), -1.0, dtype=torch.float64)
        DistTransport().exchange([plan], [snd], [rcv])
        gid_r = torch.from_numpy(sub.elem_gid[plan.recv_ids].astype(np.float64))
        ok = all(torch.equal(rcv[r], gid_r * 10 + r) for r in range(rows))
        Path(out_dir, f"rank{rank}.txt").write_text(f"{int(ok)} {plan.n_send} {plan.n_recv}")
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_dist_transport_delivers_every_ghost_gloo(tmp_path, world):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        ok, ns, nr = (tmp_path / f"rank{r}.txt").read_text().split()
        assert ok == "1" and int(ns) > 0 and int(nr) > 0


# ---------------------------------------------------------------------------------------------------------------
# End to end on CPU: two ranks (gloo), one partition each, HOST tensors through DistTransport every RK stage, with the
# oracle standing in for the kernels of each partition (its RHS on the local mesh: owned elements + one ghost layer,
# ghost outer edges closed).  What this pins without a GPU: the ghost layer is all a stage needs, the send / receive
# lists and the transport put every value where the next stage reads it, and the order of calls of
# PartitionedDgswem.step (stage -> exchange state) reproduces the undivided run.  The RK combine is numpy here (no fma),
# so the comparison with the undivided oracle is to round-off, not bitwise (bitwise is the GPU tests' job).
def _e2e_workload():
    from workloads import c3
    return c3(nn=14, nsteps=6)            # jittered, permuted, shelf bathymetry, M2 tide on the east side


def _e2e_worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from oracle import oracle as orc
    from paper_2508_21208_b200.partition import partition
    from paper_2508_21208_b200.decomp import HaloPlan, DistTransport
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        w = _e2e_workload(); m = w.mesh
        prm = dict(w.params); prm["wetdry"] = 0; prm["limiter"] = 0
        sub = partition(m.xy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, world)[rank]
        plan = HaloPlan(sub)
        o = orc.Oracle(prm, sub.xy, np.asarray(w.bathy)[sub.node_gid], sub.tri, sub.edge_elem, sub.edge_local, sub.edge_bc, sub.elem_edge)
        o.set_tide(*w.tide)
        gid = sub.elem_gid
        # a non-trivial smooth state so that every mode and every exchange matters
        rng = np.random.default_rng(7)
        full = [0.05 * rng.standard_normal((3, m.n_elem)) for _ in range(3)]
        st = [np.ascontiguousarray(f[:, gid]) for f in full]
        wet = np.ones(sub.n_local, dtype=np.uint8)
        tr = DistTransport()

        def exchange(state):
            snd = torch.from_numpy(np.concatenate([a[:, plan.send_ids] for a in state], axis=0).copy())
            rcv = torch.zeros((9, plan.n_recv), dtype=torch.float64)
            tr.exchange([plan], [snd], [rcv])
            r = rcv.numpy()
            for c in range(3):
                state[c][:, plan.recv_ids] = r[3 * c:3 * c + 3]

        t, dt = 0.0, w.dt
        for _ in range(w.nsteps):
            w0 = [a.copy() for a in st]
            for s, (a, b, cs) in enumerate(((0.0, 1.0, 0.0), (0.5, 0.5, 1.0))):      # SSP(2,2)
                o.set_state_raw(t + cs * dt, *st, wet)
                rhs = o.eval_rhs()
                st = [a * w0[c] + b * (st[c] + dt * rhs[c]) if s else st[c] + dt * rhs[c] for c in range(3)]
                exchange(st)
            t += dt
        np.save(Path(out_dir, f"state{rank}.npy"), np.stack([a[:, :sub.n_owned] for a in st]))
        np.save(Path(out_dir, f"gid{rank}.npy"), gid[:sub.n_owned])
    finally:
        dist.destroy_process_group()


def test_two_rank_decomposed_run_equals_undivided_oracle_gloo(tmp_path):
    import torch.multiprocessing as mp
    from oracle import oracle as orc
    orc.build()
    w = _e2e_workload(); m = w.mesh
    prm = dict(w.params); prm["wetdry"] = 0; prm["limiter"] = 0
    o = orc.Oracle(prm, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
    o.set_tide(*w.tide)
    rng = np.random.default_rng(7)
    full = [0.05 * rng.standard_normal((3, m.n_elem)) for _ in range(3)]
    o.set_state_raw(0.0, *full, np.ones(m.n_elem, dtype=np.uint8))
    o.step(w.nsteps, w.dt)
    _, *ref = o.get_state()
    world = 2
    mp.spawn(_e2e_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    seen = np.zeros(m.n_elem, dtype=bool)
    for r in range(world):
        st = np.load(tmp_path / f"state{r}.npy"); gid = np.load(tmp_path / f"gid{r}.npy")
        assert not seen[gid].any()
        seen[gid] = True
        for c in range(3):
            scale = np.abs(ref[c]).max()
            assert np.abs(st[c] - ref[c][:, gid]).max() <= 1e-12 * scale, (r, c)
    assert seen.all()
    # and the exchange is what makes it so: without it the ghosts go stale and the owned elements next to them drift
    assert np.abs(ref[0]).max() > 1e-3
