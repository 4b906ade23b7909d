"""TEST ONLY: builds and loads tests/hostcheck/libhostcheck.so, the CUDA path's per-tip arithmetic compiled
for the host CPU by nvcc (same headers the kernels inline).  Lets the GPU-less tier check that arithmetic
against the oracle before any GPU time is spent.  Not used by the product, the GPU tests or bench.py."""
import ctypes as C
import os
import subprocess

import numpy as np

from paper_2505_22822_b200 import binding as B

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "host_math_check.cu")
LIB = os.path.join(HERE, "libhostcheck.so")
CSRC = os.path.join(HERE, "..", "..", "paper_2505_22822_b200", "csrc")
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lib = None


def lib():
    global _lib
    if _lib is None:
        deps = [SRC] + [os.path.join(CSRC, f) for f in ("ckf_math.cuh", "ckf_nav.cuh", "ckf_host_geom.h")]
        if not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in deps):
            tmp = LIB + ".tmp.%d" % os.getpid()
            subprocess.run(["/usr/local/cuda/bin/nvcc", "-O2", "-std=c++17", "-shared", "-Xcompiler", "-fPIC",
                            "-Wno-deprecated-gpu-targets", SRC, "-o", tmp], check=True)
            os.replace(tmp, LIB)
        L = C.CDLL(LIB)
        L.hm_create.restype = C.c_void_p
        L.hm_create.argtypes = [C.POINTER(B.ckf_geometry), C.POINTER(B.ckf_field), C.POINTER(B.ckf_config)]
        L.hm_destroy.argtypes = [C.c_void_p]
        L.hm_move.restype = C.c_int
        L.hm_move.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp, _dp, _ip, _dp, _dp, _ip]
        L.hm_update.argtypes = [C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.hm_field.argtypes = [C.c_void_p, _dp, _dp]
        L.hm_field_gradient.argtypes = [C.c_void_p, _dp, _dp]
        _lib = L
    return _lib


class HostMath:
    def __init__(self, det, fld, ckf):
        self.keep = []
        g = B.make_geometry(det, self.keep)
        f = B.make_field(fld, self.keep)
        c = B.make_config(ckf, 64, 1, 1, 1, 1)
        self.ctx = lib().hm_create(C.byref(g), C.byref(f), C.byref(c))

    def move(self, precision, module, x, Cov):
        x = np.ascontiguousarray(x, np.float64)
        Cov = np.ascontiguousarray(Cov, np.float64).reshape(36)
        xp, Cp = np.zeros(6), np.zeros(36)
        tg, tr = C.c_int32(-1), C.c_int32(0)
        st = lib().hm_move(self.ctx, precision, int(module), x.ctypes.data_as(_dp), Cov.ctypes.data_as(_dp),
                           C.byref(tg), xp.ctypes.data_as(_dp), Cp.ctypes.data_as(_dp), C.byref(tr))
        return st, tg.value, xp, Cp.reshape(6, 6), tr.value

    def update(self, precision, x, Cov, loc, var):
        x = np.ascontiguousarray(x, np.float64)
        Cov = np.ascontiguousarray(Cov, np.float64).reshape(36)
        loc = np.ascontiguousarray(loc, np.float64)
        var = np.ascontiguousarray(var, np.float64)
        xo, Co, c2 = np.zeros(6), np.zeros(36), C.c_double(0)
        lib().hm_update(precision, x.ctypes.data_as(_dp), Cov.ctypes.data_as(_dp), loc.ctypes.data_as(_dp),
                        var.ctypes.data_as(_dp), xo.ctypes.data_as(_dp), Co.ctypes.data_as(_dp), C.byref(c2))
        return xo, Co.reshape(6, 6), c2.value

    def field(self, r):
        r = np.ascontiguousarray(r, np.float64)
        b = np.zeros(3)
        lib().hm_field(self.ctx, r.ctypes.data_as(_dp), b.ctypes.data_as(_dp))
        return b

    def field_gradient(self, r):
        r = np.ascontiguousarray(r, np.float64)
        g = np.zeros(9)
        lib().hm_field_gradient(self.ctx, r.ctypes.data_as(_dp), g.ctypes.data_as(_dp))
        return g.reshape(3, 3)

    def __del__(self):
        try:
            lib().hm_destroy(self.ctx)
        except Exception:
            pass
