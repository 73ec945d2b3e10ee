#!/usr/bin/env python
"""Per-phase SM cycles of the resident kernel (k_resident, config 4's shape by default).

Builds a SECOND copy of the library with -DEA_TRACE (phase clocks compiled in; the product library
has none), runs sweeps through its C ABI and prints the cycles block 0 spends per sweep in

  parity 0 | parity 1 + energy counts | energy push + cluster barrier | swap decisions | rank masks + mask tables |
  parity 1 of the sweeps that need no energies

  python paper_1311_5582_b200/examples/resident_phases.py [L] [n_temps] [n_realizations] [swap_interval]
"""
import ctypes as C
import os
import subprocess
import sys
import tempfile

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
sys.path.insert(0, os.path.dirname(PKG))
from ea_inputs import temperature_ladder  # noqa: E402


def main():
    L = int(sys.argv[1]) if len(sys.argv) > 1 else 16
    nT = int(sys.argv[2]) if len(sys.argv) > 2 else 24
    R = int(sys.argv[3]) if len(sys.argv) > 3 else 2048
    swap = int(sys.argv[4]) if len(sys.argv) > 4 else 1
    so = os.path.join(tempfile.mkdtemp(), "libea_trace.so")
    subprocess.check_call([os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"), "-gencode", "arch=compute_100a,code=sm_100a",
                           "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-shared", "-DEA_TRACE", "-o", so,
                           os.path.join(PKG, "csrc", "ea_lib.cu")])
    lib = C.CDLL(so)
    lib.ea_create.restype = C.c_void_p
    lib.ea_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_uint64]
    lib.ea_sweep.argtypes = [C.c_void_p, C.c_int64, C.c_int]
    lib.ea_synchronize.argtypes = [C.c_void_p]
    lib.ea_get_kernel.argtypes = [C.c_void_p]
    lib.ea_destroy.argtypes = [C.c_void_p]
    lib.ea_debug_res_trace.argtypes = [C.c_void_p, C.c_int]
    betas = np.ascontiguousarray(1.0 / temperature_ladder(nT, 0.7, 2.0))
    h = lib.ea_create(L, nT, R, betas.ctypes.data_as(C.c_void_p), 4)
    assert h, "ea_create failed (needs a CUDA device)"
    assert lib.ea_get_kernel(h) == 2 and L in (8, 16), "this shape does not run on k_resident"
    ns = 200
    assert lib.ea_sweep(h, ns, swap) == 0 and lib.ea_synchronize(h) == 0          # warm-up
    assert lib.ea_debug_res_trace(None, 1) == 0
    assert lib.ea_sweep(h, ns, swap) == 0 and lib.ea_synchronize(h) == 0
    out = (C.c_ulonglong * 8)()
    assert lib.ea_debug_res_trace(out, 0) == 0
    lib.ea_destroy(h)
    names = ["parity 0", "parity 1 + energy counts", "energy push + cluster barrier", "swap decisions",
             "rank masks + mask tables", "parity 1 of sweeps without a swap"]
    tot = float(sum(out[:6]))
    print(f"L={L} n_temps={nT} realizations={R} swap every {swap}: block 0, {ns} sweeps of one launch, SM cycles per sweep")
    for n, v in zip(names, out[:6]):
        print(f"  {n:32s} {v / ns:9.1f}  {100 * v / tot:5.1f} %")
    print(f"  {'whole sweep':32s} {tot / ns:9.1f}")
    print(f"  per launch: prologue (state and tables into shared memory) {out[6]} cycles, epilogue (write-back issued) {out[7]} cycles")


if __name__ == "__main__":
    main()
