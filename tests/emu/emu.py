"""TEST-ONLY ctypes wrapper of the host-emulated CUDA kernels (tests/emu/emu_driver.cpp)."""
import ctypes as C
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
LIB = os.path.join(HERE, "libark_emu.so")
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lib = None


def build():
    srcs = [os.path.join(HERE, "emu_driver.cpp"), os.path.join(HERE, "ark_emu.h"),
            os.path.join(ROOT, "paper_1903_09043_b200", "csrc", "ark_device.cuh"),
            os.path.join(ROOT, "paper_1903_09043_b200", "csrc", "ark_step.cuh"),
            os.path.join(ROOT, "paper_1903_09043_b200", "csrc", "ark_step3d.cuh")]
    if os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in srcs):
        return LIB
    subprocess.run(["g++", "-std=c++20", "-O1", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
                    "-I", HERE, "-o", LIB, srcs[0]], check=True)
    return LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.emu_run.argtypes = ([C.c_int] * 3 + [C.c_double, C.c_double, _dp, C.c_double, C.c_double, C.c_int, _ip, _dp]
                                 + [_dp] * 5 + [C.c_int, _dp, C.c_int, _dp, _dp, _dp, C.c_int, _dp])
        _lib.emu_run.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def run(prm, U, dts, zchunk=0, want_padded=False):
    """-> (U_new, rates_after_each_step, rate_of_initial_state[, padded ghost-filled initial state]).
    prm.get("energy_form") == 1 selects the Appendix-B energy update, prm.get("phi") an array-valued potential."""
    nx, ny, nz = prm["nx"], prm["ny"], prm["nz"]
    n = nx * ny * nz
    S = [np.zeros(n) if (a is None) else np.array(a, dtype=np.float64).reshape(-1).copy() for a in U]
    g = np.ascontiguousarray(prm["g"], dtype=np.float64)
    bt = np.ascontiguousarray(np.asarray(prm["bc_type"], dtype=np.int32).reshape(6))
    bv = np.ascontiguousarray(np.asarray(prm["bc_value"], dtype=np.float64).reshape(6))
    dts = np.ascontiguousarray(dts, dtype=np.float64)
    rates = np.zeros(max(len(dts), 1))
    rate0 = np.zeros(1)
    nf = 5 if nz > 1 else 4
    padded = np.zeros(nf * (nx + 4) * (ny + 4) * ((nz + 4) if nz > 1 else 1)) if want_padded else None
    phi = prm.get("phi")
    phi = None if phi is None else np.ascontiguousarray(np.asarray(phi, dtype=np.float64).reshape(-1))
    lib().emu_run(nx, ny, nz, prm["dx"], prm["gamma"], _p(g), prm["mu"], prm["kappa"], prm["theta"],
                  bt.ctypes.data_as(_ip), _p(bv), *[_p(a) for a in S], len(dts), _p(dts), int(zchunk),
                  _p(rates), _p(rate0), _p(padded), int(prm.get("energy_form", 0)), _p(phi))
    out = (S, rates[:len(dts)], float(rate0[0]))
    if want_padded:
        shp = (nf, (nz + 4) if nz > 1 else 1, ny + 4, nx + 4)
        out = out + (padded.reshape(shp),)
    return out
