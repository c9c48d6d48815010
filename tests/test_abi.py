"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/dgswem.h declares; the binding fails loudly without a device; the oracle is not on the
product path."""
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2508_21208_b200 import build, load_library
    build.build()
    return load_library()


def test_header_symbols_are_exported(lib):
    hdr = (ROOT / "include" / "dgswem.h").read_text()
    declared = set(re.findall(r"\b(dgswem_[a-z0-9_]+)\s*\(", hdr))
    assert {"dgswem_create", "dgswem_set_state", "dgswem_step", "dgswem_get_state", "dgswem_eval_rhs",
            "dgswem_get_wetdry", "dgswem_set_tide", "dgswem_set_wind_holland", "dgswem_destroy"} <= declared
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2508_21208_b200 import EXPORTS
    assert set(EXPORTS) == declared


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2508_21208_b200 import Dgswem
    from workloads import c1
    w = c1(nq=4)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        Dgswem.from_workload(w)


def test_product_does_not_touch_the_oracle():
    """Nothing under the package or include/ may import, include or link anything under oracle/."""
    for f in list((ROOT / "paper_2508_21208_b200").rglob("*")) + list((ROOT / "include").rglob("*")):
        if f.is_file() and f.suffix in (".py", ".cu", ".cuh", ".h", ".cpp"):
            txt = f.read_text()
            assert "oracle" not in txt.lower().replace("the oracle bit for bit", "").replace("with the oracle", ""), f
    for f in (ROOT / "oracle").rglob("*"):
        if f.is_file() and f.suffix in (".py", ".c", ".h"):
            txt = f.read_text()
            assert "import paper_2508_21208_b200" not in txt and "libdgswem" not in txt and "dgswem.h\"" not in txt.replace("dgswem_oracle.h\"", ""), f


def test_sass_has_fp64_and_no_float_atomics():
    """The kernels are fp64 (DADD/DMUL present) and contain no floating-point atomics (the DFMAs are
    the explicit fma() calls of the canonical arithmetic, the compiler contracts nothing by itself: -fmad=false)."""
    import shutil, subprocess
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not available")
    from paper_2508_21208_b200 import LIB_PATH
    sass = subprocess.run(["cuobjdump", "-sass", str(LIB_PATH)], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass
    body = sass[sass.index("k_elem"):]
    assert "DMUL" in body and "DADD" in body
    assert "RED." not in sass and "ATOM" not in sass


def _raw_create(lib, w, *, params=None, tri=None, edge_elem=None, edge_bc=None, elem_edge=None):
    """dgswem_create through ctypes with NULL hooks (no torch, no device memory before validation)."""
    import ctypes as C
    import numpy as np
    from paper_2508_21208_b200.binding import Params
    m = w.mesh
    prm = dict(w.params) if params is None else params
    P = Params(p=int(prm["p"]), rk_order=int(prm["rk_order"]), g=prm["g"], cf=prm["cf"], coriolis_f=prm["coriolis_f"],
               h0_dry=prm["h0_dry"], limiter=int(prm["limiter"]), wetdry=int(prm["wetdry"]), reorder=int(prm.get("reorder", 1)), device=0,
               rk_stages=int(prm.get("rk_stages", 0)))
    xy = np.ascontiguousarray(m.xy, dtype=np.float64)
    bathy = np.ascontiguousarray(w.bathy, dtype=np.float64)
    tri = np.ascontiguousarray(m.tri if tri is None else tri, dtype=np.int32)
    ee = np.ascontiguousarray(m.edge_elem if edge_elem is None else edge_elem, dtype=np.int32)
    el = np.ascontiguousarray(m.edge_local, dtype=np.int8)
    bc = np.ascontiguousarray(m.edge_bc if edge_bc is None else edge_bc, dtype=np.int32)
    eled = np.ascontiguousarray(m.elem_edge if elem_edge is None else elem_edge, dtype=np.int32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
    h = C.c_void_p()
    rc = lib.dgswem_create(C.byref(h), C.byref(P), None, xy.shape[0], dp(xy), dp(bathy), tri.shape[0], ip(tri), ee.shape[0],
                           ip(ee), el.ctypes.data_as(C.POINTER(C.c_int8)), ip(bc), ip(eled))
    msg = lib.dgswem_last_error(None)
    if rc == 0:
        lib.dgswem_destroy(h)
    return rc, (msg.decode() if msg else "")


def test_create_validates_arguments_and_mesh_on_the_host(lib):
    """Argument and mesh validation runs before any CUDA call, so its error codes can be checked here:
    -1 bad parameter, -2 inconsistent tables (orientation, edge/element cross references, boundary codes);
    a valid mesh gets as far as the device (0 with a GPU, -3 'no CUDA device' without)."""
    import numpy as np
    from workloads import c1
    w = c1(nq=4)
    m = w.mesh
    for key, val in (("p", 4), ("p", 0), ("rk_order", 4), ("rk_stages", 5), ("rk_stages", 1), ("reorder", 3), ("h0_dry", 0.0), ("h0_dry", 1e-200), ("g", -9.81), ("cf", -1.0)):
        bad = dict(w.params); bad[key] = val
        rc, msg = _raw_create(lib, w, params=bad)
        assert rc == -1, (key, val, rc, msg)
    rc, msg = _raw_create(lib, w, tri=m.tri[:, ::-1].copy())                 # clockwise elements
    assert rc == -2 and "counter-clockwise" in msg
    tri = m.tri.copy(); tri[3, 1] = m.n_nodes + 5                             # node id out of range
    assert _raw_create(lib, w, tri=tri)[0] == -2
    ee = m.edge_elem.copy(); ee[0, 0] = (ee[0, 0] + 1) % m.n_elem             # edge points at the wrong element
    assert _raw_create(lib, w, edge_elem=ee)[0] == -2
    eled = m.elem_edge.copy(); eled[2, 0], eled[2, 1] = eled[2, 1], eled[2, 0]   # local edges swapped
    assert _raw_create(lib, w, elem_edge=eled)[0] == -2
    bc = m.edge_bc.copy(); bc[np.flatnonzero(m.edge_elem[:, 1] >= 0)[0]] = 1  # interior edge with a boundary code
    assert _raw_create(lib, w, edge_bc=bc)[0] == -2
    bc = m.edge_bc.copy(); bc[np.flatnonzero(m.edge_elem[:, 1] < 0)[0]] = 0   # boundary edge without one
    assert _raw_create(lib, w, edge_bc=bc)[0] == -2
    rc, msg = _raw_create(lib, w)
    import torch
    assert rc == (0 if torch.cuda.is_available() else -3), (rc, msg)


def test_create_rejects_null_and_degenerate_sizes(lib):
    """NULL tables, an empty mesh and out-of-range sizes are argument errors (-1), found before any CUDA call."""
    import ctypes as C
    import numpy as np
    from paper_2508_21208_b200.binding import Params
    from workloads import c1
    w = c1(nq=2)
    m = w.mesh
    prm = w.params
    P = Params(p=1, rk_order=2, g=prm["g"], cf=0.0, coriolis_f=0.0, h0_dry=prm["h0_dry"], limiter=0, wetdry=0, reorder=1, device=0)
    xy = np.ascontiguousarray(m.xy); b = np.ascontiguousarray(w.bathy); tri = np.ascontiguousarray(m.tri, dtype=np.int32)
    ee = np.ascontiguousarray(m.edge_elem, dtype=np.int32); el = np.ascontiguousarray(m.edge_local, dtype=np.int8)
    bc = np.ascontiguousarray(m.edge_bc, dtype=np.int32); eled = np.ascontiguousarray(m.elem_edge, dtype=np.int32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double)); ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
    i8 = el.ctypes.data_as(C.POINTER(C.c_int8))
    h = C.c_void_p()
    full = [C.byref(h), C.byref(P), None, m.n_nodes, dp(xy), dp(b), m.n_elem, ip(tri), m.n_edge, ip(ee), i8, ip(bc), ip(eled)]
    for pos in (1, 4, 5, 7, 9, 10, 11, 12):                       # params and every table pointer
        a = list(full); a[pos] = None
        assert lib.dgswem_create(*a) == -1
    for pos, val in ((3, 2), (6, 0), (8, 2), (6, -5)):            # n_nodes < 3, n_elem < 1, n_edge < 3, negative
        a = list(full); a[pos] = val
        assert lib.dgswem_create(*a) == -1
    assert lib.dgswem_create(None, *full[1:]) == -1               # no place to put the handle
    # calls on a NULL handle are argument errors, not crashes
    assert lib.dgswem_step(None, 1, 1.0) == -1 and lib.dgswem_sync(None) == -1 and lib.dgswem_begin_step(None, 1.0) == -1
    assert lib.dgswem_launch_count(None) == 0 and lib.dgswem_stage_form(None) == 0
    lib.dgswem_destroy(None)
