"""ctypes wrapper around the ORACLE (oracle/ark_oracle.cpp).

Test infrastructure only: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  It does not import, and is
not imported by, the CUDA package paper_1903_09043_b200.
"""
import ctypes as C

import numpy as np

from . import build as _build

BC_PERIODIC, BC_REFLECTING, BC_FIXED_T, BC_FLUX = 0, 1, 2, 3

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        common = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp, C.c_double, C.c_double,
                  C.c_int, _ip, _dp]
        _lib.oracle_run.argtypes = common + [_dp] * 5 + [C.c_int, C.c_double, _dp, _dp, C.c_int]
        _lib.oracle_run.restype = C.c_int
        _lib.oracle_run_phi.argtypes = common + [_dp] * 5 + [C.c_int, C.c_double, _dp, _dp, C.c_int, _dp]
        _lib.oracle_run_phi.restype = C.c_int
        _lib.oracle_max_rate.argtypes = common + [_dp] * 5
        _lib.oracle_max_rate.restype = C.c_double
        _lib.oracle_fill_ghosts.argtypes = common + [_dp] * 10
        _lib.oracle_fill_ghosts.restype = C.c_int
        _lib.oracle_face.argtypes = [C.c_double] * 8 + [C.c_int, _dp]
        _lib.oracle_face.restype = None
        _lib.oracle_K.restype = C.c_double
        _lib.oracle_diagnostics.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp] + [_dp] * 5 + [_dp]
        _lib.oracle_diagnostics.restype = None
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _common(p):
    """p: dict with nx, ny, nz, dx, gamma, g(3), mu, kappa, theta, bc_type(3x2), bc_value(3x2)."""
    g = np.ascontiguousarray(p["g"], dtype=np.float64)
    bt = np.ascontiguousarray(np.asarray(p["bc_type"], dtype=np.int32).reshape(6))
    bv = np.ascontiguousarray(np.asarray(p.get("bc_value", np.zeros((3, 2))), dtype=np.float64).reshape(6))
    args = [int(p["nx"]), int(p["ny"]), int(p["nz"]), float(p["dx"]), float(p["gamma"]), _ptr(g),
            float(p["mu"]), float(p["kappa"]), int(p["theta"]), bt.ctypes.data_as(_ip), _ptr(bv)]
    return args, (g, bt, bv)


def _state(p, U):
    n = int(p["nx"]) * int(p["ny"]) * int(p["nz"])
    out = []
    for f in range(5):
        if f == 3 and int(p["nz"]) == 1 and (len(U) < 5 or U[3] is None):
            out.append(np.zeros(n))
            continue
        a = np.array(U[f], dtype=np.float64, order="C").reshape(-1)
        assert a.size == n, (a.size, n)
        out.append(a)
    return out


def run(p, U, nsteps, cfl=None, dts=None, form=0):
    """Advance a copy of U = [rho, rhou, rhov, rhow, E] (dense, any shape of nx*ny*nz elements,
    x fastest) by nsteps.  Either dts (array of nsteps prescribed steps) or cfl.  form: 0 = E + gravity source
    (normative), 1 = eq. (11), 2 = Appendix B (non-conservative energy); p.get("energy_form") == 1 also selects
    Appendix B.  p.get("phi"): optional dense potential at the cell centres, else Phi = -g.x.
    Returns (U_new list of flat arrays, dts_used)."""
    args, keep = _common(p)
    S = _state(p, U)
    dts_in = None if dts is None else np.ascontiguousarray(dts, dtype=np.float64)
    dts_out = np.zeros(max(nsteps, 1))
    if form == 0 and int(p.get("energy_form", 0)) == 1:
        form = 2
    phi = p.get("phi")
    phi = None if phi is None else np.ascontiguousarray(np.asarray(phi, dtype=np.float64).reshape(-1))
    assert phi is None or phi.size == S[0].size
    rc = lib().oracle_run_phi(*args, *[_ptr(a) for a in S], int(nsteps),
                              float(cfl if cfl is not None else 0.0), _ptr(dts_in), _ptr(dts_out), int(form), _ptr(phi))
    if rc != 0:
        raise FloatingPointError("oracle: non-finite CFL rate (rc=%d)" % rc)
    return S, dts_out[:nsteps]


def max_rate(p, U):
    args, keep = _common(p)
    S = _state(p, U)
    return lib().oracle_max_rate(*args, *[_ptr(a) for a in S])


def compute_dt(p, U, cfl):
    return cfl / max_rate(p, U)


def fill_ghosts(p, U):
    """Returns the 5 padded arrays shaped (nz+4 or 1, ny+4, nx+4)."""
    args, keep = _common(p)
    S = _state(p, U)
    nx, ny, nz = int(p["nx"]), int(p["ny"]), int(p["nz"])
    shp = ((nz + 4) if nz > 1 else 1, ny + 4, nx + 4)
    P = [np.zeros(shp) for _ in range(5)]
    lib().oracle_fill_ghosts(*args, *[_ptr(a) for a in S], *[_ptr(a) for a in P])
    return P


def face(gamma, rhoL, unL, pL, rhoR, unR, pR, gh=0.0, theta_flag=1):
    """-> dict(cL, cR, a, S, ustar, theta, pistar) for one face (pin P8)."""
    out = np.zeros(7)
    lib().oracle_face(gamma, rhoL, unL, pL, rhoR, unR, pR, gh, int(theta_flag), _ptr(out))
    return dict(zip(["cL", "cR", "a", "S", "ustar", "theta", "pistar"], out.tolist()))


def diagnostics(p, U):
    """-> dict(max_speed, mean_speed, kinetic_energy, max_mach, mass, total_energy), see oracle_diagnostics."""
    S = _state(p, U)
    g = np.ascontiguousarray(p["g"], dtype=np.float64)
    out = np.zeros(6)
    lib().oracle_diagnostics(int(p["nx"]), int(p["ny"]), int(p["nz"]), float(p["dx"]), float(p["gamma"]), _ptr(g),
                             *[_ptr(a) for a in S], _ptr(out))
    return dict(zip(("max_speed", "mean_speed", "kinetic_energy", "max_mach", "mass", "total_energy"), out.tolist()))


def K():
    return lib().oracle_K()


def ke_spectrum(p, U):
    """Kinetic-energy power spectrum of the horizontal middle plane (Fig. 11; the paper prints no
    formula: reading A26 of DESIGN.md).  Plane k = nz // 2, w_c = sqrt(rho) u_c; w^_c = fft2(w_c) / (nx ny) (library FFT
    as the plain definition of the discrete Fourier transform); E[kappa] = sum over the shell floor(|k~| + 1/2) == kappa
    (signed integer wavenumbers) of 1/2 sum_c |w^_c|^2.  Pinned by Parseval (sum E = plane mean of 1/2 rho |u|^2), a single
    Fourier mode in closed form and a brute-force DFT (tests/test_oracle_pins.py)."""
    nx, ny, nz = int(p["nx"]), int(p["ny"]), int(p["nz"])
    S = [a.reshape(nz, ny, nx) for a in _state(p, U)]
    k = nz // 2
    rho = S[0][k]
    power = np.zeros((ny, nx))
    for c in (1, 2, 3):
        w = S[c][k] / np.sqrt(rho)
        W = np.fft.fft2(w) / (nx * ny)
        power += 0.5 * (W.real ** 2 + W.imag ** 2)
    kx = np.fft.fftfreq(nx, 1.0 / nx)[None, :]
    ky = np.fft.fftfreq(ny, 1.0 / ny)[:, None]
    shell = np.floor(np.sqrt(kx * kx + ky * ky) + 0.5).astype(np.int64)
    nb = int(np.floor(np.sqrt((nx // 2) ** 2 + (ny // 2) ** 2) + 0.5)) + 1
    return np.bincount(shell.reshape(-1), weights=power.reshape(-1), minlength=nb)[:nb]
