"""paper_2605_31425_b200: B200-native (sm_100a) minimum-enclosing-ball solver.

Hand-written CUDA kernels behind a C-ABI shared library (``include/meb.h``,
``libmeb_b200.so``) plus a thin ctypes binding with the same names.  Importing the package
does not load the library; the first call does, and raises if it is missing -- there is no
CPU fallback and nothing here imports the CPU oracle.
"""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTS, LIB_PATH, Context, MebError, load  # noqa: F401


def build(verbose: bool = False) -> str:
    """Compile every CUDA source for sm_100a into libmeb_b200.so (in-tree).  Returns its path."""
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    res = subprocess.run(["bash", os.path.join(here, "build.sh")], capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc build of libmeb_b200.so failed")
    return LIB_PATH
