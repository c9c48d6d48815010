"""The binary32 build of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT): the source of oracle/oracle.py executed
once more with F32 on, i.e. the same ctypes wrapper over oracle/liborc32.so = dgswem_oracle.c compiled with -DORC_F32
(same expression trees, one IEEE binary32 operation per operator or fmaf call).  Arrays in and out are float32; time,
time step, tidal parameters and the storm track stay binary64 (PAPER.md:158 "-r4", :529: the paper's runs are single
precision)."""
import importlib.util
import sys
from pathlib import Path

_spec = importlib.util.spec_from_file_location("oracle._oracle32_impl", Path(__file__).resolve().parent / "oracle.py")
_mod = importlib.util.module_from_spec(_spec)
_mod._ORC_F32 = True
sys.modules["oracle._oracle32_impl"] = _mod
_spec.loader.exec_module(_mod)
globals().update({k: v for k, v in vars(_mod).items() if not k.startswith("__")})
