"""Domain-decomposed driver on top of the stage-granular C ABI.

One `Dgswem` handle per partition (`partition.py`: owned elements + one layer of ghosts), and per time step

    begin_step;  for every RK stage s:  stage_rhs(s);  [limiter on: exchange means; stage_limit(s)];  exchange state;  end_step

where an exchange is `halo_pack` on the owner, transport, `halo_unpack` on the ghost side.  Every step of the arithmetic
runs in the library's kernels; this module only orders the calls and moves the packed halo buffers:

  * `LocalTransport`: all partitions live in this process (on one GPU): device-to-device copies between the packed
    buffers.  This is what the GPU tests run: a partitioned run must reproduce the undivided run bit for bit.
  * `DistTransport`: one partition per rank of a `torch.distributed` group (NCCL between GPUs over NVLink; gloo with
    host tensors in the CPU test of the exchange plan): `batch_isend_irecv` of one contiguous slice per neighbour rank.
"""
from __future__ import annotations

import numpy as np

from .partition import partition, SubMesh


class HaloPlan:
    """Column offsets of every neighbour part in a partition's packed send / receive buffers ([rows][n])."""

    def __init__(self, sub: SubMesh):
        self.send_ids, self.recv_ids, self.peers, scnt, rcnt = sub.halo_lists()
        self.send_off, self.recv_off = {}, {}
        so = ro = 0
        for q, sc, rc in zip(self.peers, scnt, rcnt):
            self.send_off[q] = (so, sc); so += sc
            self.recv_off[q] = (ro, rc); ro += rc
        self.n_send, self.n_recv = so, ro


class LocalTransport:
    """All partitions in one process: copy each packed slice to its destination's receive buffer."""

    def exchange(self, plans, send_bufs, recv_bufs):
        for p, plan in enumerate(plans):
            for q in plan.peers:
                so, sc = plan.send_off[q]
                ro, rc = plans[q].recv_off[p]
                if sc != rc:
                    raise RuntimeError("halo plans of two partitions disagree")
                if sc:
                    recv_bufs[q][:, ro:ro + rc] = send_bufs[p][:, so:so + sc]


class DistTransport:
    """One partition per rank: one isend / irecv per neighbour rank, slices made contiguous per peer."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group)

    def exchange(self, plans, send_bufs, recv_bufs):
        # plans / buffers hold only this rank's partition, at index 0
        plan, snd, rcv = plans[0], send_bufs[0], recv_bufs[0]
        ops, stage = [], []
        for q in plan.peers:
            so, sc = plan.send_off[q]
            ro, rc = plan.recv_off[q]
            if sc:
                s = snd[:, so:so + sc].contiguous()
                ops.append(self.dist.P2POp(self.dist.isend, s, q, self.group))
            if rc:
                r = rcv.new_empty((rcv.shape[0], rc))
                stage.append((r, ro, rc))
                ops.append(self.dist.P2POp(self.dist.irecv, r, q, self.group))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()
        for r, ro, rc in stage:
            rcv[:, ro:ro + rc] = r


class PartitionedDgswem:
    """The undivided model's interface (set_state / step / get_state / get_wetdry) on a partitioned mesh.

    parts=None: this process drives every partition (LocalTransport, one GPU).  parts=[r]: this process drives partition r
    only and `transport` must be a DistTransport whose ranks are the part ids."""

    def __init__(self, params, xy, bathy, tri, edge_elem, edge_local, edge_bc, elem_edge, n_parts, *, tide=None, holland=None,
                 pressure=False, rain=0.0, precision=64,
                 reorder=1, device=0, parts=None, transport=None, part_of_element=None, overlap=None, graph=False):
        import torch
        from .binding import Dgswem
        self.torch = torch
        # the vertex-neighbourhood limiter bounds an element by the means of every element around its vertices: its
        # partitions carry all foreign elements that share a node with an owned one, not only the edge-neighbours
        self.subs = partition(xy, tri, edge_elem, edge_local, edge_bc, elem_edge, n_parts, part=part_of_element,
                              ghost="vertex" if int(params["limiter"]) == 2 else "edge")
        self.mine = list(range(n_parts)) if parts is None else list(parts)
        self.transport = transport if transport is not None else LocalTransport()
        # overlap of the exchange with the interior elements: on by default where there is a wire to hide (one partition per
        # rank); with every partition on one GPU the split only adds launches (C3, 4 partitions: 91.7 against 102.8 G DOF-updates/s)
        self.overlap = (transport is not None and not isinstance(transport, LocalTransport)) if overlap is None else bool(overlap)
        self.comm = torch.cuda.Stream(device=device)      # the transport's stream: runs beside the partitions' streams
        self.cap = torch.cuda.Stream(device=device)       # the stream a whole step is recorded on and replayed from (graph=True)
        self.graph = bool(graph)
        self._graph, self._graph_dt = None, None
        self.launches_per_graph_step = 0
        if self.graph and transport is not None and not isinstance(transport, LocalTransport):
            raise ValueError("graph=True records device copies between partitions of one process: LocalTransport only")
        self.n_elem = int(np.asarray(tri).shape[0])
        self.limiter = bool(params["limiter"])
        self.n_stage = int(params.get("rk_stages", 0)) or int(params["rk_order"])
        bathy = np.asarray(bathy, dtype=np.float64)
        self.handles, self.plans, self.sbuf, self.rbuf = [], [], [], []
        for p in self.mine:
            sm = self.subs[p]
            g = Dgswem(params, sm.xy, bathy[sm.node_gid], sm.tri, sm.edge_elem, sm.edge_local, sm.edge_bc, sm.elem_edge,
                       reorder=reorder, device=device, precision=precision)
            if tide is not None:
                g.set_tide(*tide)
            if holland is not None:
                g.set_wind_holland(holland)
                if pressure:                               # surface-pressure gradient of the vortex (R-15)
                    g.set_wind_forcing(True, True)
            elif pressure:
                raise ValueError("pressure=True needs a Holland vortex (holland=...)")
            if rain:
                g.set_rain(float(rain))                    # uniform mass source (R-16)
            plan = HaloPlan(sm)
            g.set_halo(plan.send_ids, plan.recv_ids)
            rows = g.halo_rows(0)
            dev = torch.device("cuda", device)
            self.sbuf.append(torch.empty((rows, max(plan.n_send, 1)), dtype=torch.float64, device=dev))
            self.rbuf.append(torch.empty((rows, max(plan.n_recv, 1)), dtype=torch.float64, device=dev))
            self.handles.append(g)
            self.plans.append(plan)
        self.ndof = self.handles[0].ndof
        # LocalTransport indexes plans by part id: only valid when this process drives all parts
        if parts is not None and isinstance(self.transport, LocalTransport):
            raise ValueError("driving a subset of the partitions needs a DistTransport")

    @classmethod
    def from_workload(cls, w, n_parts, **kw):
        """Every forcing the workload carries (tide, vortex, and the pressure / rain notes of workloads.with_forcing), as
        Dgswem.from_workload applies them to an undivided run, and the initial state."""
        m = w.mesh
        pd = cls(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, n_parts, tide=w.tide,
                 holland=w.holland, pressure=bool(w.notes.get("pressure")), rain=float(w.notes.get("rain") or 0.0), **kw)
        pd.set_state(0.0, w.ze, w.qx, w.qy)
        return pd

    # ------------------------------------------------------------------
    def _exchange_begin(self, what):
        """Pack on each handle's stream, then the transport on the communication stream once every pack is done."""
        rows = self.handles[0].halo_rows(what)
        # contiguous [rows][n_send] / [rows][n_recv] views of the preallocated buffers, as the library packs them
        snd = [b.view(-1)[:rows * pl.n_send].view(rows, pl.n_send) for b, pl in zip(self.sbuf, self.plans)]
        rcv = [b.view(-1)[:rows * pl.n_recv].view(rows, pl.n_recv) for b, pl in zip(self.rbuf, self.plans)]
        # stream-ordered, no host synchronisation.  (A handle's next pack comes after its unpack, which has waited for the
        # transport: the buffers are free again by then.)
        torch = self.torch
        comm = self.comm
        for g, pl, s in zip(self.handles, self.plans, snd):
            if pl.n_send:
                g.halo_pack(what, s)
            ev = torch.cuda.Event()
            ev.record(g.stream)
            comm.wait_event(ev)
        with torch.cuda.stream(comm):
            self.transport.exchange(self.plans, snd, rcv)
            done = torch.cuda.Event()
            done.record(comm)
        return rcv, done

    def _exchange_end(self, what, pending):
        """Unpack on each handle's stream once the transport is done."""
        rcv, done = pending
        for g, pl, r in zip(self.handles, self.plans, rcv):
            g.stream.wait_event(done)
            if pl.n_recv:
                g.halo_unpack(what, r)

    def _exchange(self, what):
        self._exchange_end(what, self._exchange_begin(what))

    def join(self):
        """Make torch's current stream wait for everything enqueued on the partitions' streams (for timing with events)."""
        cur = self.torch.cuda.current_stream()
        ev = self.torch.cuda.Event(); ev.record(self.cap); cur.wait_event(ev)
        for g in self.handles:
            ev = self.torch.cuda.Event()
            ev.record(g.stream)
            cur.wait_event(ev)

    def set_state(self, t, ze, qx, qy):
        for p, g in zip(self.mine, self.handles):
            gid = self.subs[p].elem_gid
            g.set_state(t, np.ascontiguousarray(ze[:, gid]), np.ascontiguousarray(qx[:, gid]), np.ascontiguousarray(qy[:, gid]))

    def _one_step(self, dt):
        for g in self.handles:
            g.begin_step(dt)
        for s in range(self.n_stage):
            first_what = 1 if self.limiter else 0           # what the stage's first exchange carries
            if self.overlap:
                for g in self.handles:
                    g.stage_rhs(s, part=1)
                pending = self._exchange_begin(first_what)
                for g in self.handles:
                    g.stage_rhs(s, part=2)
                self._exchange_end(first_what, pending)
            else:
                for g in self.handles:
                    g.stage_rhs(s)
                self._exchange(first_what)
            if self.limiter:
                for g in self.handles:
                    g.stage_limit(s)
                self._exchange(0)
        for g in self.handles:
            g.end_step()

    def step(self, nsteps, dt):
        """overlap: every stage first runs on the elements other partitions wait for (dgswem_stage_rhs_part 1), packs them and
        starts the transport on the communication stream, and only then runs on the interior elements, so that the exchange
        travels while they are computed; the unpack waits for both.
        graph (LocalTransport only): the whole step -- every partition's kernels, packs, copies, unpacks, with their event
        dependencies -- is recorded once into ONE CUDA graph (dgswem_capture_mode) and replayed; per-step scalars come
        from each handle's device table (dgswem_graph_steps).  Same bits in every mode."""
        nsteps = int(nsteps)
        if not self.graph:
            for _ in range(nsteps):
                self._one_step(dt)
            return
        torch = self.torch
        if self._graph is None or self._graph_dt != dt:
            self._capture(dt)
        done = 0
        while done < nsteps:
            n = min(nsteps - done, 4096)
            for g in self.handles:                       # scalar rows of the next n steps, on each handle's stream
                g.graph_steps(n, dt)
                ev = torch.cuda.Event(); ev.record(g.stream); self.cap.wait_event(ev)
            with torch.cuda.stream(self.cap):
                for _ in range(n):
                    self._graph.replay()
                fin = torch.cuda.Event(); fin.record(self.cap)
            for g in self.handles:                       # the next upload / any later call on a handle comes after the replays
                g.stream.wait_event(fin)
            done += n

    def _capture(self, dt):
        torch = self.torch
        torch.cuda.synchronize()
        l0 = sum(g.launch_count() for g in self.handles)
        for g in self.handles:
            g.capture_mode(True)
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=self.cap, capture_error_mode="relaxed"):
                fork = torch.cuda.Event(); fork.record(self.cap)
                for g in self.handles:                   # the handles' streams join the capture
                    g.stream.wait_event(fork)
                self.comm.wait_event(fork)
                self._one_step(dt)
                for st in [g.stream for g in self.handles] + [self.comm]:
                    ev = torch.cuda.Event(); ev.record(st); self.cap.wait_event(ev)
        finally:
            for g in self.handles:
                g.capture_mode(False)
        self._graph, self._graph_dt = graph, dt
        # kernels of the library recorded into one step of the graph (the library counts launches, recorded ones included)
        self.launches_per_graph_step = sum(g.launch_count() for g in self.handles) - l0

    def get_state(self):
        """(t, ze, qx, qy) of the elements this process owns, scattered into global-size arrays (others stay NaN)."""
        out = [np.full((self.ndof, self.n_elem), np.nan) for _ in range(3)]
        t = None
        for p, g in zip(self.mine, self.handles):
            sm = self.subs[p]
            t, *st = g.get_state()
            own = sm.elem_gid[:sm.n_owned]
            for c in range(3):
                out[c][:, own] = st[c][:, :sm.n_owned]
        return (t, *out)

    def get_wetdry(self):
        out = np.full(self.n_elem, 255, dtype=np.uint8)
        for p, g in zip(self.mine, self.handles):
            sm = self.subs[p]
            out[sm.elem_gid[:sm.n_owned]] = g.get_wetdry()[:sm.n_owned]
        return out

    def close(self):
        for g in self.handles:
            g.close()
        self.handles = []
