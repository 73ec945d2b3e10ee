#!/usr/bin/env python
"""Per-phase timing of the streaming kernel (k_stream, config 5's shape by default).

Builds a SECOND copy of the library with -DEA_TRACE (phase time stamps compiled in; the product
library has none), runs a few sweeps through its C ABI and prints, per phase, the median over the
blocks of the time spent in it (us), for sweeps 2..7 of the call:

  parity 0 | grid barrier + first tiles | parity 1 (+ energy counts) | grid barrier | swap decisions + mask tables

  python paper_1311_5582_b200/examples/stream_phases.py [L] [n_temps] [n_realizations]
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
    L = int(sys.argv[1]) if len(sys.argv) > 1 else 32
    nT = int(sys.argv[2]) if len(sys.argv) > 2 else 32
    R = int(sys.argv[3]) if len(sys.argv) > 3 else 256
    tmp = tempfile.mkdtemp()
    so, trace = os.path.join(tmp, "libea_trace.so"), os.path.join(tmp, "trace.bin")
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
    betas = np.ascontiguousarray(1.0 / temperature_ladder(nT, 0.9, 2.0))
    h = lib.ea_create(L, nT, R, betas.ctypes.data_as(C.c_void_p), 5)
    assert h, "ea_create failed (needs a CUDA device)"
    assert lib.ea_get_kernel(h) == 4, "this shape does not run on the streaming kernel"
    assert lib.ea_sweep(h, 50, 1) == 0 and lib.ea_synchronize(h) == 0        # warm-up, untraced
    os.environ["EA_STREAM_TRACE"] = trace
    assert lib.ea_sweep(h, 8, 1) == 0 and lib.ea_synchronize(h) == 0
    del os.environ["EA_STREAM_TRACE"]
    lib.ea_destroy(h)
    t = np.fromfile(trace, dtype=np.uint64).reshape(-1, 8, 8).astype(np.float64)     # [block][sweep][stamp] ns
    t = t[:, 2:, :6]
    names = ["parity 0", "grid barrier + first tiles", "parity 1 (+ energy counts)", "grid barrier",
             "swap decisions + mask tables"]
    d = np.diff(t, axis=2) / 1e3
    print(f"L={L} n_temps={nT} realizations={R}: {t.shape[0]} blocks, sweeps 2..7 of a call (us)")
    for i, n in enumerate(names):
        x = d[:, :, i]
        print(f"  {n:32s} median {np.median(x):6.2f}   min {x.min():6.2f}   max {x.max():6.2f}")
    per_sweep = (t[:, 1:, 0] - t[:, :-1, 0]) / 1e3
    print(f"  {'whole sweep':32s} median {np.median(per_sweep):6.2f}")
    spread1 = (t[:, :, 1].max(axis=0) - t[:, :, 1].min(axis=0)) / 1e3
    spread3 = (t[:, :, 3].max(axis=0) - t[:, :, 3].min(axis=0)) / 1e3
    print(f"  spread between blocks at the end of parity 0 / parity 1: {np.median(spread1):.2f} / {np.median(spread3):.2f}")


if __name__ == "__main__":
    main()
