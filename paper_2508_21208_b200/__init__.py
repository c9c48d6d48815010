"""B200-native hot path of DG-SWEM's explicit time step (arxiv 2508.21208).

`Dgswem` is the ctypes binding of the C-ABI library `libdgswem.so` (include/dgswem.h), whose
sm_100a fp64 CUDA kernels do all the work.  Build the library in-tree with
`python -m paper_2508_21208_b200.build`.
"""
from .binding import Dgswem, DgswemError, load_library, LIB_PATH, EXPORTS, nodal_static  # noqa: F401
