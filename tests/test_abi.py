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
    declared = set(re.findall(r"\b(dgswem_[a-z_]+)\s*\(", hdr))
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
    """The kernels are fp64 (DADD/DMUL present) and contain no floating-point atomics or FMA
    contractions."""
    import shutil, subprocess
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not available")
    from paper_2508_21208_b200 import LIB_PATH
    sass = subprocess.run(["cuobjdump", "-sass", str(LIB_PATH)], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass
    body = sass[sass.index("k_elem"):]
    assert "DMUL" in body and "DADD" in body
    assert "RED." not in sass and "ATOM" not in sass
