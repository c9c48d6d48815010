"""ctypes binding of libdgswem.so (include/dgswem.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; this module converts numpy
arrays to pointers, backs the library's device allocations with torch tensors and hands it torch's
current CUDA stream.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "libdgswem.so"

E_NONFINITE = -4


class Params(C.Structure):
    _fields_ = [("p", C.c_int32), ("rk_order", C.c_int32), ("g", C.c_double), ("cf", C.c_double),
                ("coriolis_f", C.c_double), ("h0_dry", C.c_double), ("limiter", C.c_int32), ("wetdry", C.c_int32),
                ("reorder", C.c_int32), ("device", C.c_int32), ("flux", C.c_int32), ("precision", C.c_int32),
                ("rk_stages", C.c_int32)]


class Holland(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("x0", "y0", "vx", "vy", "rmax", "dp", "B", "rho_air", "rho_water", "f")]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class DevHooks(C.Structure):
    _fields_ = [("alloc", ALLOC_FN), ("free", FREE_FN), ("user", C.c_void_p), ("stream", C.c_void_p)]


class DgswemError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dgswem error {code}: {msg}")
        self.code = code


EXPORTS = ["dgswem_create", "dgswem_set_state", "dgswem_set_tide", "dgswem_set_wind_holland", "dgswem_set_wind_forcing", "dgswem_set_rain", "dgswem_get_pressure", "dgswem_step",
           "dgswem_eval_rhs", "dgswem_get_flux", "dgswem_get_state", "dgswem_get_wetdry", "dgswem_get_nodal", "dgswem_get_wind",
           "dgswem_begin_step", "dgswem_stage_rhs", "dgswem_stage_rhs_part", "dgswem_stage_limit", "dgswem_end_step", "dgswem_capture_mode", "dgswem_graph_steps", "dgswem_set_halo",
           "dgswem_halo_pack", "dgswem_halo_unpack", "dgswem_test_math", "dgswem_fp64_peak", "dgswem_stage_form", "dgswem_precision", "dgswem_launch_count", "dgswem_profile", "dgswem_profile_read", "dgswem_sync", "dgswem_last_error", "dgswem_destroy",
           "dgswem_nodal_static", "dgswem_nodal_static_error"]

_lib = None


def load_library():
    """dlopen the in-tree library (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2508_21208_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    D, I64, VP = C.c_double, C.c_int64, C.c_void_p
    PD, PI32 = C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.dgswem_create.argtypes = [C.POINTER(VP), C.POINTER(Params), C.POINTER(DevHooks), I64, PD, PD, I64, PI32, I64, PI32,
                                C.POINTER(C.c_int8), PI32, PI32]
    L.dgswem_create.restype = C.c_int
    L.dgswem_set_state.argtypes = [VP, D, PD, PD, PD]
    L.dgswem_set_tide.argtypes = [VP, D, D, D]
    L.dgswem_set_wind_holland.argtypes = [VP, C.POINTER(Holland)]
    L.dgswem_set_wind_forcing.argtypes = [VP, C.c_int, C.c_int]
    L.dgswem_set_rain.argtypes = [VP, D]
    L.dgswem_get_pressure.argtypes = [VP, PD]
    L.dgswem_step.argtypes = [VP, I64, D]
    L.dgswem_eval_rhs.argtypes = [VP, PD, PD, PD]
    L.dgswem_get_flux.argtypes = [VP, PD]
    L.dgswem_get_state.argtypes = [VP, PD, PD, PD, PD]
    L.dgswem_get_wetdry.argtypes = [VP, C.POINTER(C.c_uint8)]
    L.dgswem_get_wind.argtypes = [VP, PD]
    L.dgswem_get_nodal.argtypes = [VP, PD, PD, PD]
    L.dgswem_test_math.argtypes = [VP, I64, PD, PD]
    L.dgswem_begin_step.argtypes = [VP, D]
    L.dgswem_stage_rhs.argtypes = [VP, C.c_int]
    L.dgswem_stage_rhs_part.argtypes = [VP, C.c_int, C.c_int]
    L.dgswem_stage_limit.argtypes = [VP, C.c_int]
    L.dgswem_end_step.argtypes = [VP]
    L.dgswem_capture_mode.argtypes = [VP, C.c_int]
    L.dgswem_graph_steps.argtypes = [VP, I64, D]
    L.dgswem_set_halo.argtypes = [VP, I64, PI32, I64, PI32]
    L.dgswem_halo_pack.argtypes = [VP, C.c_int, C.c_void_p, C.c_int]
    L.dgswem_halo_unpack.argtypes = [VP, C.c_int, C.c_void_p, C.c_int]
    L.dgswem_fp64_peak.argtypes = [VP, PD]; L.dgswem_fp64_peak.restype = C.c_int
    L.dgswem_stage_form.argtypes = [VP]; L.dgswem_stage_form.restype = C.c_int
    L.dgswem_precision.argtypes = [VP]; L.dgswem_precision.restype = C.c_int
    L.dgswem_launch_count.argtypes = [VP]; L.dgswem_launch_count.restype = I64
    L.dgswem_profile.argtypes = [VP, C.c_int]; L.dgswem_profile.restype = C.c_int
    L.dgswem_profile_read.argtypes = [VP, PD, C.POINTER(I64)]; L.dgswem_profile_read.restype = C.c_int
    L.dgswem_sync.argtypes = [VP]
    L.dgswem_last_error.argtypes = [VP]; L.dgswem_last_error.restype = C.c_char_p
    L.dgswem_destroy.argtypes = [VP]; L.dgswem_destroy.restype = None
    L.dgswem_nodal_static.argtypes = [C.c_int, VP, C.c_int, I64, I64, VP, VP, VP, VP, VP, VP, VP]; L.dgswem_nodal_static.restype = C.c_int
    L.dgswem_nodal_static_error.argtypes = []; L.dgswem_nodal_static_error.restype = C.c_char_p
    for name in ("dgswem_set_state", "dgswem_set_tide", "dgswem_set_wind_holland", "dgswem_set_wind_forcing", "dgswem_set_rain",
                 "dgswem_get_pressure", "dgswem_step", "dgswem_eval_rhs",
                 "dgswem_get_flux", "dgswem_get_state", "dgswem_get_wetdry", "dgswem_get_wind", "dgswem_sync",
                 "dgswem_begin_step", "dgswem_stage_rhs", "dgswem_stage_rhs_part", "dgswem_stage_limit", "dgswem_end_step", "dgswem_capture_mode", "dgswem_graph_steps", "dgswem_set_halo",
                 "dgswem_halo_pack", "dgswem_halo_unpack", "dgswem_test_math", "dgswem_get_nodal"):
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


STATIC_MAX_ELEM = 524288     # DGSWEM_STATIC_MAX_ELEM / DGSWEM_STATIC_MAX_NODES of include/dgswem.h
STATIC_MAX_NODES = 524288


def nodal_static(p, tri, ze, qx, qy, zn, qxn, qyn, *, n_nodes=None, n_elem=None):
    """dgswem_nodal_static: element-averaged nodal values of a modal state, for callers that cannot
    allocate device memory when they need them (a stream capture is open, a memory pool owns the GPU, the time loop
    must not stall on cudaMalloc): no handle, no allocation -- the node -> element table is rebuilt per call in the
    library's fixed 20 MiB device array, hence the limits STATIC_MAX_ELEM / STATIC_MAX_NODES (DgswemError beyond them).

    Every argument is a contiguous torch CUDA tensor owned by the caller, all on one device: tri int32 [n_elem, 3];
    ze, qx, qy float64 [ndof, n_elem]; outputs zn, qxn, qyn float64 [n_nodes], overwritten.  Kernels are enqueued on
    torch's current stream of that device; nothing is synchronised.  Same bits as Dgswem.get_nodal for the same mesh
    and state.  Make the first call on a device outside any stream capture, and do not let two calls overlap on one GPU
    (they share the array).  n_nodes / n_elem override the sizes taken from the tensor shapes (tests of the limits)."""
    import torch
    ts = (tri, ze, qx, qy, zn, qxn, qyn)
    dev = tri.device
    if dev.type != "cuda" or any(t.device != dev for t in ts):
        raise ValueError("nodal_static takes CUDA tensors on one device (there is no CPU fallback)")
    if any(not t.is_contiguous() for t in ts):
        raise ValueError("nodal_static takes contiguous tensors")
    if tri.dtype != torch.int32 or any(t.dtype != torch.float64 for t in ts[1:]):
        raise ValueError("tri must be int32, all other tensors float64")
    ndof = (int(p) + 1) * (int(p) + 2) // 2
    ne = tri.shape[0] if n_elem is None else int(n_elem)
    nn = zn.shape[0] if n_nodes is None else int(n_nodes)
    if n_elem is None and n_nodes is None:
        if tri.shape != (ne, 3) or any(t.shape != (ndof, ne) for t in (ze, qx, qy)) or any(t.shape != (nn,) for t in (zn, qxn, qyn)):
            raise ValueError("shapes: tri [n_elem, 3]; ze, qx, qy [ndof, n_elem]; zn, qxn, qyn [n_nodes]")
    L = load_library()
    idx = dev.index if dev.index is not None else torch.cuda.current_device()
    rc = L.dgswem_nodal_static(idx, torch.cuda.current_stream(dev).cuda_stream, int(p), nn, ne,
                               *(t.data_ptr() for t in ts))
    if rc != 0:
        raise DgswemError(rc, (L.dgswem_nodal_static_error() or b"").decode())


class Dgswem:
    """One model on one GPU.  Method names mirror the C ABI (dgswem_<name>)."""

    def __init__(self, params: dict, xy, bathy, tri, edge_elem, edge_local, edge_bc, elem_edge, *,
                 reorder: int = 1, device: int = 0, use_torch_alloc: bool = True, precision: int = 64):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2508_21208_b200 needs a CUDA device (there is no CPU fallback)")
        L = load_library()
        self.L = L
        self.p = int(params["p"])
        self.ndof = (self.p + 1) * (self.p + 2) // 2
        self.nqe = self.p + 1
        self.n_stage = int(params.get("rk_stages", 0)) or int(params["rk_order"])
        xy = np.ascontiguousarray(xy, dtype=np.float64)
        bathy = np.ascontiguousarray(bathy, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        edge_elem = np.ascontiguousarray(edge_elem, dtype=np.int32)
        edge_local = np.ascontiguousarray(edge_local, dtype=np.int8)
        edge_bc = np.ascontiguousarray(edge_bc, dtype=np.int32)
        elem_edge = np.ascontiguousarray(elem_edge, dtype=np.int32)
        self.n_nodes, self.n_elem, self.n_edge = xy.shape[0], tri.shape[0], edge_elem.shape[0]
        assert xy.shape == (self.n_nodes, 2) and bathy.shape == (self.n_nodes,) and tri.shape == (self.n_elem, 3)
        assert edge_elem.shape == (self.n_edge, 2) and edge_local.shape == (self.n_edge, 2)
        assert edge_bc.shape == (self.n_edge,) and elem_edge.shape == (self.n_elem, 3)
        prm = Params(p=self.p, rk_order=int(params["rk_order"]), rk_stages=int(params.get("rk_stages", 0)), g=params["g"], cf=params["cf"], coriolis_f=params["coriolis_f"],
                     h0_dry=params["h0_dry"], limiter=int(params["limiter"]), wetdry=int(params["wetdry"]),
                     reorder=int(reorder), device=int(device), flux=int(params.get("flux", 0)),
                     precision=int(precision))
        self.device = torch.device("cuda", device)
        self._tensors = {}
        self.stream = None
        hooks = None
        if use_torch_alloc:
            def _alloc(nbytes, _user):
                try:
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
                except Exception:
                    return None
                self._tensors[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, _user):
                self._tensors.pop(ptr, None)

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)   # keep the callbacks alive
            # a dedicated (non-default) torch stream per handle: all kernels and copies of this model run
            # on it; time it with torch.cuda.Event(...).record(model.stream)
            self.stream = torch.cuda.Stream(device=self.device)
            hooks = DevHooks(self._alloc_cb, self._free_cb, None, C.c_void_p(self.stream.cuda_stream))
        self.h = C.c_void_p()
        i32 = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        rc = L.dgswem_create(C.byref(self.h), C.byref(prm), C.byref(hooks) if hooks is not None else None,
                             self.n_nodes, _dp(xy), _dp(bathy), self.n_elem, i32(tri), self.n_edge, i32(edge_elem),
                             edge_local.ctypes.data_as(C.POINTER(C.c_int8)), i32(edge_bc), i32(elem_edge))
        if rc != 0:
            msg = L.dgswem_last_error(None)
            self.h = None
            raise DgswemError(rc, msg.decode() if msg else "?")

    @classmethod
    def from_workload(cls, w, **kw):
        m = w.mesh
        o = cls(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge, **kw)
        if w.tide is not None:
            o.set_tide(*w.tide)
        if w.holland is not None:
            o.set_wind_holland(w.holland)
            if w.notes.get("pressure"):
                o.set_wind_forcing(True, True)
        if w.notes.get("rain"):
            o.set_rain(w.notes["rain"])
        o.set_state(0.0, w.ze, w.qx, w.qy)
        return o

    # ------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            msg = self.L.dgswem_last_error(self.h)
            raise DgswemError(rc, msg.decode() if msg else "?")

    def _st(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.shape != (self.ndof, self.n_elem):
            raise ValueError(f"state array must be [{self.ndof}, {self.n_elem}], got {a.shape}")
        return a

    def set_state(self, t, ze, qx, qy):
        ze, qx, qy = self._st(ze), self._st(qx), self._st(qy)
        self._check(self.L.dgswem_set_state(self.h, float(t), _dp(ze), _dp(qx), _dp(qy)))

    def set_tide(self, amp, omega, phase):
        self._check(self.L.dgswem_set_tide(self.h, float(amp), float(omega), float(phase)))

    def set_wind_holland(self, hol: dict | None):
        if hol is None:
            self._check(self.L.dgswem_set_wind_holland(self.h, None))
        else:
            self._check(self.L.dgswem_set_wind_holland(self.h, C.byref(Holland(**hol))))

    def set_wind_forcing(self, stress=True, pressure=False):
        self._check(self.L.dgswem_set_wind_forcing(self.h, int(bool(stress)), int(bool(pressure))))

    def set_rain(self, rate):
        self._check(self.L.dgswem_set_rain(self.h, float(rate)))

    def step(self, nsteps, dt):
        self._check(self.L.dgswem_step(self.h, int(nsteps), float(dt)))

    def eval_rhs(self):
        r = [np.empty((self.ndof, self.n_elem)) for _ in range(3)]
        self._check(self.L.dgswem_eval_rhs(self.h, *[_dp(a) for a in r]))
        return r

    def get_flux(self):
        f = np.empty((3, self.nqe, self.n_edge))
        self._check(self.L.dgswem_get_flux(self.h, _dp(f)))
        return f

    def get_state(self, out=None):
        if out is None:
            out = [np.empty((self.ndof, self.n_elem)) for _ in range(3)]
        t = C.c_double()
        self._check(self.L.dgswem_get_state(self.h, C.byref(t), *[_dp(a) for a in out]))
        return (t.value, *out)

    def get_wetdry(self):
        wet = np.empty(self.n_elem, dtype=np.uint8)
        self._check(self.L.dgswem_get_wetdry(self.h, wet.ctypes.data_as(C.POINTER(C.c_uint8))))
        return wet

    def get_nodal(self):
        """Element-averaged nodal values: [zeta, Qx, Qy], each [n_nodes]."""
        out = [np.empty(self.n_nodes) for _ in range(3)]
        self._check(self.L.dgswem_get_nodal(self.h, *[_dp(a) for a in out]))
        return out

    def get_wind(self):
        tau = np.empty((2, self.n_nodes))
        self._check(self.L.dgswem_get_wind(self.h, _dp(tau)))
        return tau

    def get_pressure(self):
        ep = np.empty(self.n_nodes)
        self._check(self.L.dgswem_get_pressure(self.h, _dp(ep)))
        return ep

    # ---- stage-granular stepping and halo lists (domain decomposition building blocks)
    def begin_step(self, dt):
        self._check(self.L.dgswem_begin_step(self.h, float(dt)))

    def stage_rhs(self, s, part=0):
        """part = 0: the whole mesh; 1: the send-list elements only; 2: all the others (dgswem_stage_rhs_part)."""
        if part:
            self._check(self.L.dgswem_stage_rhs_part(self.h, int(s), int(part)))
        else:
            self._check(self.L.dgswem_stage_rhs(self.h, int(s)))

    def capture_mode(self, on):
        self._check(self.L.dgswem_capture_mode(self.h, int(bool(on))))

    def graph_steps(self, nsteps, dt):
        self._check(self.L.dgswem_graph_steps(self.h, int(nsteps), float(dt)))

    def stage_limit(self, s):
        self._check(self.L.dgswem_stage_limit(self.h, int(s)))

    def end_step(self):
        self._check(self.L.dgswem_end_step(self.h))

    def set_halo(self, send_ids, recv_ids):
        snd = np.ascontiguousarray(send_ids, dtype=np.int32)
        rcv = np.ascontiguousarray(recv_ids, dtype=np.int32)
        self.n_send, self.n_recv = snd.size, rcv.size
        i32 = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        self._check(self.L.dgswem_set_halo(self.h, snd.size, i32(snd), rcv.size, i32(rcv)))

    def halo_rows(self, what):
        return 3 * self.ndof if what == 0 else 3

    def halo_pack(self, what, buf):
        """buf: torch CUDA tensor (asynchronous on the handle's stream) or numpy array, [rows][n_send] float64."""
        if isinstance(buf, np.ndarray):
            self._check(self.L.dgswem_halo_pack(self.h, int(what), C.c_void_p(buf.ctypes.data), 0))
        else:
            self._check(self.L.dgswem_halo_pack(self.h, int(what), C.c_void_p(buf.data_ptr()), 1))

    def halo_unpack(self, what, buf):
        if isinstance(buf, np.ndarray):
            self._check(self.L.dgswem_halo_unpack(self.h, int(what), C.c_void_p(buf.ctypes.data), 0))
        else:
            self._check(self.L.dgswem_halo_unpack(self.h, int(what), C.c_void_p(buf.data_ptr()), 1))

    def test_math(self, x):
        """TEST HOOK: (rcp_rn(x), sqrt_rn(x), 1.0/x, sqrt(x)) evaluated by the device routines."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        out = np.empty((4, x.size))
        self._check(self.L.dgswem_test_math(self.h, C.c_int64(x.size), _dp(x), _dp(out)))
        return out

    def fp64_peak(self) -> float:
        """MEASUREMENT HOOK: the device's DFMA rate (thread-level DFMAs per second) from the library's probe kernel."""
        out = C.c_double()
        self._check(self.L.dgswem_fp64_peak(self.h, C.byref(out)))
        return out.value

    def precision(self) -> int:
        """Working precision of the handle: 64 or 32."""
        return int(self.L.dgswem_precision(self.h))

    def stage_form(self) -> int:
        """0: edge kernel + element kernel (flux buffer); 1: element-centric stage kernel."""
        return int(self.L.dgswem_stage_form(self.h))

    def launch_count(self) -> int:
        return int(self.L.dgswem_launch_count(self.h))

    KERNEL_KINDS = ("wind", "edge", "elem", "limwd")

    def profile(self, enable: bool):
        self._check(self.L.dgswem_profile(self.h, int(bool(enable))))

    def profile_read(self) -> dict:
        """{kind: (total_ms, launches)} since the last read."""
        ms = (C.c_double * 4)()
        cnt = (C.c_int64 * 4)()
        self._check(self.L.dgswem_profile_read(self.h, ms, cnt))
        return {k: (ms[i], int(cnt[i])) for i, k in enumerate(self.KERNEL_KINDS)}

    def sync(self):
        self._check(self.L.dgswem_sync(self.h))

    def close(self):
        if getattr(self, "h", None):
            self.L.dgswem_destroy(self.h)
            self.h = None
            self._tensors.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
