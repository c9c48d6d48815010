"""ctypes wrapper of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It builds oracle/dgswem_oracle.c with gcc (-O2
-ffp-contract=off, OpenMP) into oracle/liborc.so and exposes it 1:1.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
SRC = HERE / "dgswem_oracle.c"
HDR = HERE / "dgswem_oracle.h"
# working precision of this module instance: binary64, or binary32 when loaded through oracle/oracle32.py (-DORC_F32 build
# of the same source; arrays in and out are then float32, time / tide / storm-track scalars stay Python floats = binary64)
F32 = bool(globals().get("_ORC_F32", False))
REAL = C.c_float if F32 else C.c_double
NP = np.float32 if F32 else np.float64
LIB = HERE / ("liborc32.so" if F32 else "liborc.so")

MAXDOF, MAXQA, MAXQE = 10, 12, 4


def build(force: bool = False) -> Path:
    """Compile the oracle (idempotent)."""
    if (not force and LIB.exists() and LIB.stat().st_mtime >= max(SRC.stat().st_mtime, HDR.stat().st_mtime)):
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["gcc", "-std=c99"] + (["-DORC_F32"] if F32 else []) + ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", str(tmp), str(SRC), "-lm"]
    # fma() calls become one instruction where the CPU has it (same result: fma is correctly rounded either way)
    try:
        if " fma " in Path("/proc/cpuinfo").read_text().split("flags", 1)[1].split("\n", 1)[0] + " ":
            cmd.insert(1, "-mfma")
    except (OSError, IndexError):
        pass
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


class Params(C.Structure):
    _fields_ = [("p", C.c_int32), ("rk_order", C.c_int32), ("g", REAL), ("cf", REAL),
                ("coriolis_f", REAL), ("h0_dry", REAL), ("limiter", C.c_int32), ("wetdry", C.c_int32),
                ("flux", C.c_int32), ("rk_stages", C.c_int32)]


class Holland(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("x0", "y0", "vx", "vy", "rmax", "dp", "B", "rho_air", "rho_water", "f")]


class Tables(C.Structure):
    _fields_ = [("p", C.c_int32), ("ndof", C.c_int32), ("nqe", C.c_int32), ("nqa", C.c_int32),
                ("ge", REAL * MAXQE), ("we", REAL * MAXQE),
                ("elam", (REAL * 2) * MAXQE),
                ("la", (REAL * 3) * MAXQA), ("wa", REAL * MAXQA),
                ("invM", REAL * MAXDOF),
                ("phiA", (REAL * MAXDOF) * MAXQA),
                ("dphiA1", (REAL * MAXDOF) * MAXQA),
                ("dphiA2", (REAL * MAXDOF) * MAXQA),
                ("phiE", ((REAL * MAXDOF) * MAXQE) * 3),
                ("wfac", (REAL * MAXDOF) * MAXQA),
                ("srfac", (REAL * MAXDOF) * MAXQA),
                ("efac", ((REAL * MAXDOF) * MAXQE) * 3),
                ("phiV", (REAL * MAXDOF) * 3)]

    def np(self, name):
        return np.ctypeslib.as_array(getattr(self, name)).copy()


RHS_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_int, C.c_double, C.POINTER(REAL), C.POINTER(REAL))
POST_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_int, C.POINTER(REAL))

_lib = None


def _dp(a):
    assert a.dtype == NP, a.dtype
    return a.ctypes.data_as(C.POINTER(REAL))


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(str(build()))
    # R = working precision (`real`), D = binary64 scalars that stay binary64 in every build (time, dt, tide, storm centre)
    R, D, I32, I64, VP = REAL, C.c_double, C.c_int32, C.c_int64, C.c_void_p
    PR = C.POINTER(REAL)
    L.orc_basis.argtypes = [R, R, R, PR, PR, PR]
    L.orc_make_tables.argtypes = [C.c_int, C.POINTER(Tables)]
    L.orc_llf_flux.argtypes = [R] * 11 + [C.c_int, R, PR, PR, PR]
    L.orc_roe_flux.argtypes = [R] * 11 + [C.c_int, R, PR, PR, PR]
    L.orc_det_exp.argtypes = [R]; L.orc_det_exp.restype = R
    L.orc_det_log.argtypes = [R]; L.orc_det_log.restype = R
    L.orc_holland_node.argtypes = [C.POINTER(Holland), D, D, R, R, PR, PR, PR]
    L.orc_holland_node_p.argtypes = [C.POINTER(Holland), R, D, D, R, R, PR, PR, PR, PR]
    L.orc_limit_var.argtypes = [C.c_int, PR, PR, C.POINTER(C.c_int)]; L.orc_limit_var.restype = R
    L.orc_limit_var_vertex.argtypes = [C.c_int, PR, PR, PR]; L.orc_limit_var_vertex.restype = R
    L.orc_wetdry_elem.argtypes = [C.POINTER(Tables), R, PR, PR, PR, PR]; L.orc_wetdry_elem.restype = C.c_int
    L.orc_ssprk_step.argtypes = [C.c_int, I64, PR, PR, PR, D, D, RHS_FN, POST_FN, VP]; L.orc_ssprk_step.restype = C.c_int
    L.orc_ssprk_step_s.argtypes = [C.c_int, C.c_int, I64, PR, PR, PR, D, D, RHS_FN, POST_FN, VP]; L.orc_ssprk_step_s.restype = C.c_int
    L.orc_create.argtypes = [C.POINTER(Params), I64, PR, PR, I64, C.POINTER(I32), I64, C.POINTER(I32),
                             C.POINTER(C.c_int8), C.POINTER(I32), C.POINTER(I32)]
    L.orc_create.restype = VP
    L.orc_destroy.argtypes = [VP]
    L.orc_get_tables.argtypes = [VP]; L.orc_get_tables.restype = C.POINTER(Tables)
    L.orc_set_state.argtypes = [VP, D, PR, PR, PR]
    L.orc_set_state_raw.argtypes = [VP, D, PR, PR, PR, C.POINTER(C.c_uint8)]
    L.orc_apply_post.argtypes = [VP, C.c_int, C.c_int]
    L.orc_set_tide.argtypes = [VP, D, D, D]
    L.orc_set_wind_holland.argtypes = [VP, C.POINTER(Holland)]
    L.orc_set_wind_forcing.argtypes = [VP, C.c_int, C.c_int]
    L.orc_set_rain.argtypes = [VP, R]
    L.orc_get_pressure.argtypes = [VP, PR]
    L.orc_step.argtypes = [VP, I64, D]
    L.orc_eval_rhs.argtypes = [VP, PR, PR, PR, PR, PR, PR]
    L.orc_get_flux.argtypes = [VP, PR]
    L.orc_get_state.argtypes = [VP, C.POINTER(C.c_double), PR, PR, PR]
    L.orc_get_wetdry.argtypes = [VP, C.POINTER(C.c_uint8)]
    L.orc_get_geometry.argtypes = [VP, PR, PR, PR, PR, PR]
    L.orc_get_wind.argtypes = [VP, PR]
    L.orc_get_nodal.argtypes = [VP, PR, PR, PR]
    L.orc_get_nodal.restype = None
    L.orc_num_threads.restype = C.c_int
    _lib = L
    return L


# ------------------------------------------------------------------ piece-level helpers
def basis(lam0, lam1, lam2):
    phi, d1, d2 = (np.zeros(MAXDOF, dtype=NP) for _ in range(3))
    lib().orc_basis(lam0, lam1, lam2, _dp(phi), _dp(d1), _dp(d2))
    return phi, d1, d2


def tables(p: int) -> Tables:
    T = Tables()
    assert lib().orc_make_tables(p, C.byref(T)) == 0
    return T


def llf_flux(g, h0, nx, ny, hq, wp, wm, bc=0, zeta_b=0.0):
    out = [REAL() for _ in range(3)]
    lib().orc_llf_flux(g, h0, nx, ny, hq, wp[0], wp[1], wp[2], wm[0], wm[1], wm[2], bc, zeta_b,
                       *[C.byref(o) for o in out])
    return np.array([o.value for o in out])


def roe_flux(g, h0, nx, ny, hq, wp, wm, bc=0, zeta_b=0.0):
    out = [REAL() for _ in range(3)]
    lib().orc_roe_flux(g, h0, nx, ny, hq, wp[0], wp[1], wp[2], wm[0], wm[1], wm[2], bc, zeta_b,
                       *[C.byref(o) for o in out])
    return np.array([o.value for o in out])


def det_exp(x):
    return lib().orc_det_exp(float(x))


def det_log(x):
    return lib().orc_det_log(float(x))


def holland_node(hol: dict, cx, cy, x, y):
    h = Holland(**hol)
    out = [REAL() for _ in range(3)]
    lib().orc_holland_node(C.byref(h), cx, cy, x, y, *[C.byref(o) for o in out])
    return tuple(o.value for o in out)   # tsx, tsy, V


def holland_node_p(hol: dict, g, cx, cy, x, y):
    h = Holland(**hol)
    out = [REAL() for _ in range(4)]
    lib().orc_holland_node_p(C.byref(h), g, cx, cy, x, y, *[C.byref(o) for o in out])
    return tuple(o.value for o in out)   # tsx, tsy, V, eta_p


def limit_var(p, w, mean_nb, has_nb):
    w = np.array(w, dtype=NP)
    mn = np.array(mean_nb, dtype=NP)
    hs = (C.c_int * 3)(*[int(h) for h in has_nb])
    alpha = lib().orc_limit_var(p, _dp(w), _dp(mn), hs)
    return alpha, w


def limit_var_vertex(p, w, vmin, vmax):
    w = np.array(w, dtype=NP)
    lo = np.array(vmin, dtype=NP); hi = np.array(vmax, dtype=NP)
    alpha = lib().orc_limit_var_vertex(p, _dp(w), _dp(lo), _dp(hi))
    return alpha, w


def wetdry_elem(p, h0, hv, ze, qx, qy):
    T = tables(p)
    hv = np.array(hv, dtype=NP)
    ze, qx, qy = (np.array(a, dtype=NP) for a in (ze, qx, qy))
    wet = lib().orc_wetdry_elem(C.byref(T), h0, _dp(hv), _dp(ze), _dp(qx), _dp(qy))
    return wet, ze, qx, qy


def ssprk_step(order, w, t, dt, rhs_py, post_py=None, stages=0):
    """One SSP-RK step with a Python RHS rhs_py(stage, t_stage, w)->array; stages = 0: as many as the order."""
    w = np.array(w, dtype=NP)
    n = w.size
    w0, rhs = np.zeros(n, dtype=NP), np.zeros(n, dtype=NP)

    def _rhs(ctx, stage, ts, wp, rp):
        wa = np.ctypeslib.as_array(wp, shape=(n,))
        ra = np.ctypeslib.as_array(rp, shape=(n,))
        ra[:] = rhs_py(stage, ts, wa)

    def _post(ctx, stage, wp):
        if post_py is not None:
            wa = np.ctypeslib.as_array(wp, shape=(n,))
            post_py(stage, wa)

    rc = lib().orc_ssprk_step_s(order, stages, n, _dp(w), _dp(w0), _dp(rhs), t, dt, RHS_FN(_rhs), POST_FN(_post), None)
    assert rc == 0
    return w


# ------------------------------------------------------------------ model
class Oracle:
    """The CPU oracle of one model instance (same call names as the C-ABI of the product)."""

    def __init__(self, params: dict, xy, bathy, tri, edge_elem, edge_local, edge_bc, elem_edge):
        L = lib()
        self.L = L
        self.prm = Params(**{k: params[k] for k in ("p", "rk_order", "g", "cf", "coriolis_f", "h0_dry", "limiter", "wetdry")},
                          flux=int(params.get("flux", 0)), rk_stages=int(params.get("rk_stages", 0)))
        self.p = params["p"]
        self.ndof = (self.p + 1) * (self.p + 2) // 2
        self.nqe = self.p + 1
        xy = np.ascontiguousarray(xy, dtype=NP)
        bathy = np.ascontiguousarray(bathy, dtype=NP)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        edge_elem = np.ascontiguousarray(edge_elem, dtype=np.int32)
        edge_local = np.ascontiguousarray(edge_local, dtype=np.int8)
        edge_bc = np.ascontiguousarray(edge_bc, dtype=np.int32)
        elem_edge = np.ascontiguousarray(elem_edge, dtype=np.int32)
        self.n_nodes, self.n_elem, self.n_edge = xy.shape[0], tri.shape[0], edge_elem.shape[0]
        i32 = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        self.h = L.orc_create(C.byref(self.prm), self.n_nodes, _dp(xy), _dp(bathy), self.n_elem, i32(tri),
                              self.n_edge, i32(edge_elem), edge_local.ctypes.data_as(C.POINTER(C.c_int8)),
                              i32(edge_bc), i32(elem_edge))
        if not self.h:
            raise RuntimeError("orc_create failed")

    @classmethod
    def from_workload(cls, w):
        m = w.mesh
        o = cls(w.params, m.xy, w.bathy, m.tri, m.edge_elem, m.edge_local, m.edge_bc, m.elem_edge)
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

    def close(self):
        if self.h:
            self.L.orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def tables(self) -> Tables:
        return self.L.orc_get_tables(self.h).contents

    def _chk(self, a):
        a = np.ascontiguousarray(a, dtype=NP)
        assert a.shape == (self.ndof, self.n_elem), a.shape
        return a

    def set_state(self, t, ze, qx, qy):
        ze, qx, qy = self._chk(ze), self._chk(qx), self._chk(qy)
        self.L.orc_set_state(self.h, float(t), _dp(ze), _dp(qx), _dp(qy))

    def set_state_raw(self, t, ze, qx, qy, wet):
        """Test hook: state and wet flags as given, no initial wet/dry pass."""
        ze, qx, qy = self._chk(ze), self._chk(qx), self._chk(qy)
        wet = np.ascontiguousarray(wet, dtype=np.uint8)
        assert wet.shape == (self.n_elem,)
        self.L.orc_set_state_raw(self.h, float(t), _dp(ze), _dp(qx), _dp(qy), wet.ctypes.data_as(C.POINTER(C.c_uint8)))

    def apply_post(self, limiter=True, wetdry=True):
        """Test hook: the post-stage sequence SLOPELIM -> WETDRY on the current state."""
        self.L.orc_apply_post(self.h, int(bool(limiter)), int(bool(wetdry)))

    def set_tide(self, amp, omega, phase):
        self.L.orc_set_tide(self.h, amp, omega, phase)

    def set_wind_holland(self, hol: dict | None):
        if hol is None:
            self.L.orc_set_wind_holland(self.h, None)
        else:
            self.L.orc_set_wind_holland(self.h, C.byref(Holland(**hol)))

    def set_wind_forcing(self, stress=True, pressure=False):
        self.L.orc_set_wind_forcing(self.h, int(bool(stress)), int(bool(pressure)))

    def set_rain(self, rate):
        self.L.orc_set_rain(self.h, float(rate))

    def get_pressure(self):
        p = np.zeros(self.n_nodes, dtype=NP)
        self.L.orc_get_pressure(self.h, _dp(p))
        return p

    def step(self, nsteps, dt):
        self.L.orc_step(self.h, int(nsteps), float(dt))

    def eval_rhs(self, with_scale=False):
        shp = (self.ndof, self.n_elem)
        r = [np.zeros(shp, dtype=NP) for _ in range(3)]
        if with_scale:
            s = [np.zeros(shp, dtype=NP) for _ in range(3)]
            self.L.orc_eval_rhs(self.h, *[_dp(a) for a in r], *[_dp(a) for a in s])
            return r, s
        self.L.orc_eval_rhs(self.h, *[_dp(a) for a in r], None, None, None)
        return r

    def get_flux(self):
        f = np.zeros((3, self.nqe, self.n_edge), dtype=NP)
        self.L.orc_get_flux(self.h, _dp(f))
        return f

    def get_state(self):
        shp = (self.ndof, self.n_elem)
        ze, qx, qy = np.zeros(shp, dtype=NP), np.zeros(shp, dtype=NP), np.zeros(shp, dtype=NP)
        t = C.c_double()
        self.L.orc_get_state(self.h, C.byref(t), _dp(ze), _dp(qx), _dp(qy))
        return t.value, ze, qx, qy

    def get_wetdry(self):
        wet = np.zeros(self.n_elem, dtype=np.uint8)
        self.L.orc_get_wetdry(self.h, wet.ctypes.data_as(C.POINTER(C.c_uint8)))
        return wet

    def get_geometry(self):
        area = np.zeros(self.n_elem, dtype=NP); jinv = np.zeros((4, self.n_elem), dtype=NP); lfac = np.zeros((3, self.n_elem), dtype=NP)
        enx = np.zeros(self.n_edge, dtype=NP); eny = np.zeros(self.n_edge, dtype=NP)
        self.L.orc_get_geometry(self.h, _dp(area), _dp(jinv), _dp(lfac), _dp(enx), _dp(eny))
        return area, jinv, lfac, enx, eny

    def get_nodal(self):
        out = [np.zeros(self.n_nodes, dtype=NP) for _ in range(3)]
        self.L.orc_get_nodal(self.h, *[_dp(a) for a in out])
        return out

    def get_wind(self):
        tau = np.zeros((2, self.n_nodes), dtype=NP)
        self.L.orc_get_wind(self.h, _dp(tau))
        return tau


def num_threads() -> int:
    return lib().orc_num_threads()
