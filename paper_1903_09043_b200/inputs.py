"""Seeded synthetic inputs shaped like the paper's test cases.

This module serves BOTH the oracle tests and the CUDA path and therefore holds none of the
method's arithmetic (no fluxes, no update, no CFL): only initial states and solver parameters.
It imports neither oracle/ nor the CUDA binding.

Randomness is a stateless counter-based generator: u = mix64(seed, counter) >> 11 scaled by 2^-53,
counter = cell_index * ncomp + comp, cell_index = i + nx*(j + ny*k).  Any cell can therefore be
regenerated on its own (used by the full-size sampled-parity tests), and the same integer code runs
on numpy (host) and on torch tensors (device) with bit-identical results.

Every builder returns (params, U): params is the dict understood by both `oracle.ark_oracle` and
`paper_1903_09043_b200.binding.Solver`; U = [rho, rhou, rhov, rhow, E] dense arrays of shape
(nz, ny, nx) (x fastest), rhow = None in 2D.
"""
import math

import numpy as np

BC_PERIODIC, BC_REFLECTING, BC_FIXED_T, BC_FLUX = 0, 1, 2, 3


# --------------------------------------------------------------------------- random numbers
def _i64(v):
    """python int -> value representable as a signed 64-bit two's complement constant."""
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


_GOLD = _i64(0x9E3779B97F4A7C15)
_M1 = _i64(0xBF58476D1CE4E5B9)
_M2 = _i64(0x94D049BB133111EB)


def _lsr(x, s):
    """logical shift right of int64 two's-complement words (numpy or torch)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def uniform01(seed, counter):
    """counter: int64 array (numpy) or tensor (torch).  Returns float64 in [0,1), same container.
    splitmix64-style finaliser of (seed * GOLD + counter * GOLD + GOLD) in wrapping 64-bit arithmetic."""
    is_np = isinstance(counter, np.ndarray)
    if is_np:
        old = np.seterr(over="ignore")
    try:
        z = counter * _GOLD + _i64((int(seed) * 0x9E3779B97F4A7C15 + 0x9E3779B97F4A7C15) * 0xD1342543DE82EF95)
        z = (z ^ _lsr(z, 30)) * _M1
        z = (z ^ _lsr(z, 27)) * _M2
        z = z ^ _lsr(z, 31)
        m = _lsr(z, 11)
    finally:
        if is_np:
            np.seterr(**old)
    if is_np:
        return m.astype(np.float64) * (2.0 ** -53)
    import torch
    return m.to(torch.float64) * (2.0 ** -53)


def _cell_index(nx, ny, nz, device=None, box=None):
    """int64 cell indices i + nx*(j + ny*k) shaped (nz,ny,nx) (or the sub-box [(k0,k1),(j0,j1),(i0,i1)])."""
    (k0, k1), (j0, j1), (i0, i1) = box if box is not None else ((0, nz), (0, ny), (0, nx))
    if device is None:
        i = np.arange(i0, i1, dtype=np.int64)[None, None, :]
        j = np.arange(j0, j1, dtype=np.int64)[None, :, None]
        k = np.arange(k0, k1, dtype=np.int64)[:, None, None]
    else:
        import torch
        i = torch.arange(i0, i1, dtype=torch.int64, device=device)[None, None, :]
        j = torch.arange(j0, j1, dtype=torch.int64, device=device)[None, :, None]
        k = torch.arange(k0, k1, dtype=torch.int64, device=device)[:, None, None]
    return i + nx * (j + ny * k)


def _noise(seed, nx, ny, nz, ncomp, comp, device=None, box=None):
    """(2U-1) in [-1,1) for component comp of every cell (or of the cells of `box`)."""
    c = _cell_index(nx, ny, nz, device, box) * ncomp + comp
    return 2.0 * uniform01(seed, c) - 1.0


def _col(a, axis, device=None):
    """1-D numpy profile -> broadcastable (nz,ny,nx) array along `axis` (0:x, 1:y, 2:z)."""
    shape = [1, 1, 1]
    shape[2 - axis] = a.size
    a = np.asarray(a, dtype=np.float64).reshape(shape)
    if device is None:
        return a
    import torch
    return torch.from_numpy(a.copy()).to(device)


# --------------------------------------------------------------------------- hydrostatic columns
def hydrostatic_column(T, rho0, dphi):
    """Discrete hydrostatic balance (14), PAPER.md:237 / 372-376, as an INITIALISATION recipe
    (reading A19): p_{j+1}-p_j = -1/2 (rho_j+rho_{j+1}) dphi with p = rho T  =>
    rho_{j+1} = rho_j (T_j - dphi/2) / (T_{j+1} + dphi/2).  T: cell-centre temperatures bottom->top,
    dphi = Phi_{j+1}-Phi_j = |g| h."""
    T = np.asarray(T, dtype=np.float64)
    rho = np.empty_like(T)
    rho[0] = rho0
    for j in range(T.size - 1):
        rho[j + 1] = rho[j] * (T[j] - 0.5 * dphi) / (T[j + 1] + 0.5 * dphi)
    return rho


def polytrope(n, h, T_top, beta, m, gmag=1.0):
    """Conductive polytropic layer of depth n*h: T(z) = T_top + beta (L - z),
    rho(z0) = (T(z0)/T_top)^m at the bottom cell centre, then recursion (14) upward."""
    z = (np.arange(n) + 0.5) * h
    T = T_top + beta * (n * h - z)
    rho = hydrostatic_column(T, (T[0] / T_top) ** m, gmag * h)
    return T, rho


# --------------------------------------------------------------------------- parameter helper
def make_params(nx, ny, nz, dx, gamma, g=(0.0, 0.0, 0.0), mu=0.0, kappa=0.0, theta=1,
                bc_type=((0, 0), (0, 0), (0, 0)), bc_value=((0.0, 0.0), (0.0, 0.0), (0.0, 0.0))):
    return dict(nx=int(nx), ny=int(ny), nz=int(nz), dx=float(dx), gamma=float(gamma),
                g=tuple(float(x) for x in g), mu=float(mu), kappa=float(kappa), theta=int(theta),
                bc_type=tuple(tuple(int(v) for v in r) for r in bc_type),
                bc_value=tuple(tuple(float(v) for v in r) for r in bc_value))


def _energy(gamma, rho, u, v, w, p):
    ke = 0.5 * rho * (u * u + v * v + (w * w if w is not None else 0.0))
    return p / (gamma - 1.0) + ke


def _full(x, nx, ny, nz, device=None):
    """broadcast-materialise to a dense (nz,ny,nx) float64 array."""
    if device is None:
        return np.ascontiguousarray(np.broadcast_to(x, (nz, ny, nx)), dtype=np.float64)
    import torch
    if not isinstance(x, torch.Tensor):
        x = torch.as_tensor(x, dtype=torch.float64, device=device)
    return x.expand(nz, ny, nx).contiguous()


# --------------------------------------------------------------------------- the five BASELINE configs
def config1_atmosphere(n=128, seed=1001, amp=1e-3, theta=1, device=None):
    """BASELINE config 1: 2D n x n isothermal atmosphere rho=p=exp(-y) on [0,1]^2,
    gamma=1.4, g=(0,-1), periodic x, reflecting y, inviscid; density perturbed by amp*(2U-1) at fixed p.
    amp=0 gives the exactly balanced state of pin P3."""
    h = 1.0 / n
    gamma = 1.4
    T = np.ones(n)
    rho_c = hydrostatic_column(T, math.exp(-0.5 * h), h)
    p_c = rho_c * T
    rho = _full(_col(rho_c, 1, device), n, n, 1, device)
    p = _full(_col(p_c, 1, device), n, n, 1, device)
    if amp != 0.0:
        rho = rho * (1.0 + amp * _noise(seed, n, n, 1, 1, 0, device))
    zero = rho * 0.0
    E = p / (gamma - 1.0)
    prm = make_params(n, n, 1, h, gamma, g=(0.0, -1.0, 0.0), theta=theta,
                      bc_type=((BC_PERIODIC, BC_PERIODIC), (BC_REFLECTING, BC_REFLECTING), (0, 0)))
    return prm, [rho, zero, zero.clone() if device is not None else zero.copy(), None, E]


def config2_gresho(n=512, mach=1e-3, theta=1, device=None):
    """BASELINE config 2: Gresho vortex on [0,1]^2, rho0=1, p0=1/(gamma Ma^2),
    centre (1/2,1/2), periodic, no gravity (reading A17).  Deterministic (no seed)."""
    h = 1.0 / n
    gamma = 1.4
    xc = (np.arange(n) + 0.5) * h - 0.5
    X, Y = np.meshgrid(xc, xc, indexing="xy")            # shape (ny, nx), x fastest
    r = np.sqrt(X * X + Y * Y)
    p0 = 1.0 / (gamma * mach * mach)
    ut = np.where(r < 0.2, 5.0 * r, np.where(r < 0.4, 2.0 - 5.0 * r, 0.0))
    rs = np.maximum(r, 1e-300)
    p = np.where(r < 0.2, p0 + 12.5 * r * r,
                 np.where(r < 0.4, p0 + 12.5 * r * r + 4.0 - 20.0 * r + 4.0 * np.log(5.0 * rs),
                          p0 - 2.0 + 4.0 * math.log(2.0)))
    u = -ut * Y / rs
    v = ut * X / rs
    rho = np.ones_like(r)
    E = _energy(gamma, rho, u, v, None, p)
    U = [a.reshape(1, n, n) for a in (rho, rho * u, rho * v)] + [None, E.reshape(1, n, n)]
    if device is not None:
        import torch
        U = [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in U]
    prm = make_params(n, n, 1, h, gamma, theta=theta)
    return prm, U


def _rb_mu_kappa(gamma, m, T_top, T_bot, rho_mid, Ra, Pr, g=1.0, L=1.0):
    """Boussinesq mid-layer Rayleigh number: Ra = g (beta-beta_ad) L^4 rho_m^2 c_p/(T_m mu kappa),
    Pr = mu c_p / kappa  ->  mu, kappa.  Workload parameters, not parity targets."""
    cp = gamma / (gamma - 1.0)
    beta = g / (m + 1.0)
    beta_ad = g / cp
    Tm = 0.5 * (T_top + T_bot)
    mu2 = g * (beta - beta_ad) * L ** 4 * rho_mid ** 2 * cp * Pr / (Tm * Ra * cp)
    mu = math.sqrt(mu2)
    return mu, mu * cp / Pr


def config3_rb2d(nx=1024, ny=512, seed=1003, amp=1e-4, theta=1, device=None):
    """BASELINE config 3: 2D Rayleigh-Benard near onset: gamma=5/3, g=(0,-1), m=1.3,
    chi=1.1, Ra = 1.1 Ra_c (rigid-rigid 1707.76), Pr=1, fixed-T no-slip walls in y, periodic x,
    temperature perturbed by amp*(2U-1) at fixed rho.  Domain [0, nx/ny] x [0,1]."""
    h = 1.0 / ny
    gamma = 5.0 / 3.0
    m, chi = 1.3, 1.1
    beta = 1.0 / (m + 1.0)
    T_top = beta / (chi ** (1.0 / m) - 1.0)
    T_bot = T_top + beta
    Tc, rho_c = polytrope(ny, h, T_top, beta, m)
    rho_mid = ((0.5 * (T_top + T_bot)) / T_top) ** m
    mu, kappa = _rb_mu_kappa(gamma, m, T_top, T_bot, rho_mid, 1.1 * 1707.76, 1.0)
    rho = _full(_col(rho_c, 1, device), nx, ny, 1, device)
    T = _full(_col(Tc, 1, device), nx, ny, 1, device)
    if amp != 0.0:
        T = T * (1.0 + amp * _noise(seed, nx, ny, 1, 1, 0, device))
    p = rho * T
    zero = rho * 0.0
    E = p / (gamma - 1.0)
    prm = make_params(nx, ny, 1, h, gamma, g=(0.0, -1.0, 0.0), mu=mu, kappa=kappa, theta=theta,
                      bc_type=((BC_PERIODIC, BC_PERIODIC), (BC_FIXED_T, BC_FIXED_T), (0, 0)),
                      bc_value=((0, 0), (T_bot, T_top), (0, 0)))
    return prm, [rho, zero, zero.clone() if device is not None else zero.copy(), None, E]


def _convection3d(n, nz, m, chi, mu, kappa, wall, amp, seed, theta, device, box=None, heat=0.0):
    """3D polytropic layer under g=(0,0,-1), periodic x/y, `wall` in z, velocity noise amp*(2U-1) per
    component.  box = ((k0,k1),(j0,j1),(i0,i1)) returns only that sub-box of the state (params stay global).
    heat > 0: the bottom wall becomes an imposed-flux wall feeding heat x (conductive flux kappa*beta)."""
    h = 1.0 / nz
    gamma = 5.0 / 3.0
    beta = 1.0 / (m + 1.0)
    T_top = beta / (chi ** (1.0 / m) - 1.0)
    T_bot = T_top + beta
    Tc, rho_c = polytrope(nz, h, T_top, beta, m)
    (k0, k1), (j0, j1), (i0, i1) = box if box is not None else ((0, nz), (0, n), (0, n))
    bx, by, bz = i1 - i0, j1 - j0, k1 - k0
    rho = _full(_col(rho_c[k0:k1], 2, device), bx, by, bz, device)
    p = _full(_col((rho_c * Tc)[k0:k1], 2, device), bx, by, bz, device)
    vel = [amp * _noise(seed, n, n, nz, 3, c, device, box) for c in range(3)]
    E = _energy(gamma, rho, vel[0], vel[1], vel[2], p)
    bottom, vbot = (BC_FLUX, heat * kappa * beta) if heat > 0.0 else (wall, T_bot)
    prm = make_params(n, n, nz, h, gamma, g=(0.0, 0.0, -1.0), mu=mu, kappa=kappa, theta=theta,
                      bc_type=((BC_PERIODIC, BC_PERIODIC), (BC_PERIODIC, BC_PERIODIC), (bottom, wall)),
                      bc_value=((0, 0), (0, 0), (vbot, T_top)))
    return prm, [rho, rho * vel[0], rho * vel[1], rho * vel[2], E]


def config4_rb3d(n=256, seed=1004, amp=1e-3, theta=1, device=None, box=None):
    """BASELINE config 4: 3D turbulent Rayleigh-Benard shape: m=0.1, chi=1.1, Ra=1e6, Pr=1,
    fixed-T walls in z, velocity noise 1e-3.  mu, kappa from the mid-layer Ra (7.473e-4, 1.8683e-3)."""
    gamma, m, chi = 5.0 / 3.0, 0.1, 1.1
    beta = 1.0 / (m + 1.0)
    T_top = beta / (chi ** (1.0 / m) - 1.0)
    T_bot = T_top + beta
    rho_mid = ((0.5 * (T_top + T_bot)) / T_top) ** m
    mu, kappa = _rb_mu_kappa(gamma, m, T_top, T_bot, rho_mid, 1.0e6, 1.0)
    return _convection3d(n, n, m, chi, mu, kappa, BC_FIXED_T, amp, seed, theta, device, box)


def config5_convection3d(n=512, seed=1005, amp=1e-2, theta=1, device=None, box=None, heat=10.0):
    """BASELINE config 5: steep polytrope (m=1, chi=100), mu=1e-4, kappa=2.5e-4, heated from below at `heat` = 10 x the
    conductive flux kappa*beta through an imposed-flux bottom wall (reading A22), reflecting (insulating)
    top wall, velocity noise 1e-2.  heat=0 gives reflecting walls on both sides."""
    return _convection3d(n, n, 1.0, 100.0, 1.0e-4, 2.5e-4, BC_REFLECTING, amp, seed, theta, device, box, heat=heat)


def inviscid_convection3d(n=512, seed=1005, amp=1e-2, theta=1, device=None, box=None):
    """Measurement workload (bench.py `inviscid3d_512`): the config-5 stratification and noise WITHOUT dissipation
    (mu = kappa = 0, reflecting walls on both z sides), i.e. the Euler part of the scheme alone: the 3D step kernel's
    <VISC=0> instantiation, 80 B per cell update."""
    return _convection3d(n, n, 1.0, 100.0, 0.0, 0.0, BC_REFLECTING, amp, seed, theta, device, box, heat=0.0)


def config4_rb3d_phi(n=256, seed=1004, amp=1e-3, theta=1, device=None):
    """Measurement workload (bench.py `config4_256_phi`): BASELINE config 4 with its constant gravity g = (0,0,-1) handed
    over as the array-valued potential Phi = -g.x at the cell centres: the general path of the step kernel
    (88 B per cell update: the potential is read as a sixth field)."""
    prm, U = config4_rb3d(n, seed=seed, amp=amp, theta=theta, device=device)
    zc = (np.arange(n) + 0.5) * prm["dx"]
    prm = dict(prm, phi=_full(_col(zc, 2, device), n, n, n, device))
    return prm, U


# --------------------------------------------------------------------------- second workloads
def rayleigh_taylor(nx=200, ny=600, C=0.01, theta=1, mu=0.0, device=None):
    """Rayleigh-Taylor test case: domain [-0.25,0.25] x [-0.75,0.75] (L_x = 0.5, L_y = 1.5), rho = 1
    for y < 0 and 2 for y >= 0, u = 0, v = C/4 (1 + cos(2 pi x / L_x)) (1 + cos(2 pi y / L_y)), C = 0.01, resolution
    200 x 600.  The printed pressure "p = rho g y" is an abbreviation (it would be negative on one side): reading A23
    takes the classical setup p = p0 + rho g_y y with g = (0, -0.1), p0 = 2.5, gamma = 1.4, periodic x, reflecting y
    walls, for which the C = 0 state satisfies the discrete balance (14) exactly, as PAPER.md:421 states."""
    if ny * 0.5 / nx != 1.5:
        raise ValueError("rayleigh_taylor: the domain is 0.5 x 1.5, so ny must be 3 nx")
    h = 0.5 / nx
    gamma, gy, p0 = 1.4, -0.1, 2.5
    x = -0.25 + (np.arange(nx) + 0.5) * h
    y = -0.75 + (np.arange(ny) + 0.5) * h
    rho_c = np.where(y < 0.0, 1.0, 2.0)
    p_c = p0 + rho_c * gy * y
    rho = _full(_col(rho_c, 1, device), nx, ny, 1, device)
    p = _full(_col(p_c, 1, device), nx, ny, 1, device)
    vx = _col(1.0 + np.cos(2.0 * np.pi * x / 0.5), 0, device)
    vy = _col(1.0 + np.cos(2.0 * np.pi * y / 1.5), 1, device)
    v = _full((0.25 * C) * vx * vy, nx, ny, 1, device)
    zero = rho * 0.0
    E = _energy(gamma, rho, zero, v, None, p)
    prm = make_params(nx, ny, 1, h, gamma, g=(0.0, gy, 0.0), mu=mu, theta=theta,
                      bc_type=((BC_PERIODIC, BC_PERIODIC), (BC_REFLECTING, BC_REFLECTING), (0, 0)))
    return prm, [rho, zero, rho * v, None, E]


def rb2d_chi21(nx=128, ny=128, seed=1021, amp=1e-4, theta=1, ra_over_rac=10.0, device=None):
    """Strongly stratified 2D Rayleigh-Benard case: density ratio chi = 21 across the layer (m = 1.3,
    gamma = 5/3, g = (0,-1)), polytrope initialised by recursion (14), the temperature flux imposed on the
    bottom boundary (here the conductive flux kappa beta of the polytrope, so the unperturbed state is
    steady), fixed temperature at the top, periodic x.  mu, kappa from a mid-layer Rayleigh number ra_over_rac x 1707.76
    at Pr = 1 (the paper prints none: workload parameters)."""
    h = 1.0 / ny
    gamma = 5.0 / 3.0
    m, chi = 1.3, 21.0
    beta = 1.0 / (m + 1.0)
    T_top = beta / (chi ** (1.0 / m) - 1.0)
    T_bot = T_top + beta
    Tc, rho_c = polytrope(ny, h, T_top, beta, m)
    rho_mid = ((0.5 * (T_top + T_bot)) / T_top) ** m
    mu, kappa = _rb_mu_kappa(gamma, m, T_top, T_bot, rho_mid, ra_over_rac * 1707.76, 1.0)
    rho = _full(_col(rho_c, 1, device), nx, ny, 1, device)
    T = _full(_col(Tc, 1, device), nx, ny, 1, device)
    if amp != 0.0:
        T = T * (1.0 + amp * _noise(seed, nx, ny, 1, 1, 0, device))
    p = rho * T
    zero = rho * 0.0
    prm = make_params(nx, ny, 1, h, gamma, g=(0.0, -1.0, 0.0), mu=mu, kappa=kappa, theta=theta,
                      bc_type=((BC_PERIODIC, BC_PERIODIC), (BC_FLUX, BC_FIXED_T), (0, 0)),
                      bc_value=((0, 0), (kappa * beta, T_top), (0, 0)))
    return prm, [rho, zero, zero.clone() if device is not None else zero.copy(), None, p / (gamma - 1.0)]


# --------------------------------------------------------------------------- extra test problems
def sod_tube(nx=100, ny=4, theta=1):
    """Sod shock tube along x on [0,1], reflecting x walls, periodic y (reading A16)."""
    h = 1.0 / nx
    gamma = 1.4
    x = (np.arange(nx) + 0.5) * h
    rho = np.where(x < 0.5, 1.0, 0.125)
    p = np.where(x < 0.5, 1.0, 0.1)
    rho = np.ascontiguousarray(np.broadcast_to(rho, (1, ny, nx)))
    p = np.ascontiguousarray(np.broadcast_to(p, (1, ny, nx)))
    prm = make_params(nx, ny, 1, h, gamma, theta=theta,
                      bc_type=((BC_REFLECTING, BC_REFLECTING), (BC_PERIODIC, BC_PERIODIC), (0, 0)))
    return prm, [rho, np.zeros_like(rho), np.zeros_like(rho), None, p / (gamma - 1.0)]


def random_state(nx, ny, nz, seed, gamma=1.4, g=(0.0, 0.0, 0.0), mu=0.0, kappa=0.0, theta=1,
                 bc_type=((0, 0), (0, 0), (0, 0)), bc_value=((0, 0), (0, 0), (0, 0)), h=None, vel=0.3):
    """Generic smooth-free random state (rho in [0.5,1.5], p in [0.5,1.5], |u_d| < vel) for structural tests."""
    h = 1.0 / max(nx, ny, nz) if h is None else h
    nc = 5
    rho = 1.0 + 0.5 * _noise(seed, nx, ny, nz, nc, 0)
    p = 1.0 + 0.5 * _noise(seed, nx, ny, nz, nc, 1)
    u = vel * _noise(seed, nx, ny, nz, nc, 2)
    v = vel * _noise(seed, nx, ny, nz, nc, 3)
    w = vel * _noise(seed, nx, ny, nz, nc, 4) if nz > 1 else None
    E = _energy(gamma, rho, u, v, w, p)
    prm = make_params(nx, ny, nz, h, gamma, g=g, mu=mu, kappa=kappa, theta=theta, bc_type=bc_type, bc_value=bc_value)
    return prm, [rho, rho * u, rho * v, (rho * w if w is not None else None), E]
