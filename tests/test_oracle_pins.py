"""Pins for the ORACLE (oracle/ark_oracle.cpp): it is checked against what the paper and the mathematics fix,
never against itself or the CUDA path.  P-numbers follow SURVEY.md 8(c) / DESIGN.md.  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import ark_oracle as O
from paper_1903_09043_b200 import inputs as I

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PER, REF, FIX = I.BC_PERIODIC, I.BC_REFLECTING, I.BC_FIXED_T


def prim(prm, S):
    g = prm["gamma"]
    rho = S[0]
    u, v, w = S[1] / rho, S[2] / rho, S[3] / rho
    p = (g - 1.0) * (S[4] - 0.5 * rho * (u * u + v * v + w * w))
    return rho, u, v, w, p


# ----------------------------------------------------------------------------------------------- P8
def test_P8_hand_computed_face():
    """Sod left/right states through PAPER.md:152 and eq. (13), K=1.1: values worked by hand
    in tests/golden/face_sod.txt."""
    vals = {}
    for line in open(os.path.join(GOLDEN, "face_sod.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            vals[k] = float(v)
    f = O.face(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, gh=0.0, theta_flag=1)
    for k, v in vals.items():
        assert abs(f[k] - v) < 5e-10 * max(1.0, abs(v)), (k, f[k], v)
    # independent re-derivation with python floats
    cL, cR = math.sqrt(1.4), math.sqrt(1.4 * 0.1 / 0.125)
    a = O.K() * max(cL, 0.125 * cR)
    us = 0.9 / (2 * a)
    assert abs(f["ustar"] - us) < 1e-15 and abs(f["theta"] - us / cL) < 1e-15
    # theta disabled -> 1 ; moving states: sign of the upwinding term in Pi*
    f1 = O.face(1.4, 1.0, 0.3, 1.0, 1.0, -0.2, 1.0, theta_flag=0)
    a1 = O.K() * math.sqrt(1.4)
    assert f1["theta"] == 1.0
    assert abs(f1["ustar"] - 0.05) < 1e-15                     # equal pressures: plain average
    assert abs(f1["pistar"] - (1.0 + 0.5 * a1 * 0.5)) < 1e-15  # compression raises Pi*
    # gravity term: hydrostatic pair p_R - p_L = S  =>  u* = 0 exactly representable case
    f2 = O.face(1.4, 1.0, 0.0, 1.0, 1.0, 0.0, 0.5, gh=-0.5, theta_flag=1)
    assert f2["S"] == -0.5 and f2["ustar"] == 0.0 and f2["pistar"] == 0.75


# ----------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("shape", [(8, 6, 1), (6, 5, 7)])
def test_P1_uniform_state_is_bit_exact(shape):
    """g=0, uniform state: u*=u, Pi*=p, every bracket exactly 0, L~=1."""
    nx, ny, nz = shape
    prm = I.make_params(nx, ny, nz, 0.1, 1.4, mu=0.01, kappa=0.02)
    rho, u, v, w, p = 1.25, 0.5, -0.25, (0.125 if nz > 1 else 0.0), 0.75
    E = p / 0.4 + 0.5 * rho * (u * u + v * v + w * w)
    U = [np.full(shape[::-1], x) for x in (rho, rho * u, rho * v, rho * w, E)]
    S, _ = O.run(prm, U, 5, cfl=0.4)
    for f in range(5):
        assert np.array_equal(S[f], U[f].reshape(-1)), f


# ----------------------------------------------------------------------------------------------- P2
def _totals(prm, S, shape):
    nx, ny, nz = prm["nx"], prm["ny"], prm["nz"]
    h = prm["dx"]
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    Phi = -(prm["g"][0] * (i + 0.5) * h + prm["g"][1] * (j + 0.5) * h + prm["g"][2] * (k + 0.5) * h).reshape(-1)
    return [math.fsum(S[0]), math.fsum(S[1]), math.fsum(S[2]), math.fsum(S[3]), math.fsum(S[4] + S[0] * Phi)]


@pytest.mark.parametrize("case", ["periodic2d", "periodic3d", "gravity_walls2d", "gravity_walls3d", "viscous_walls3d"])
def test_P2_conservation(case):
    """Machine-precision conservation of mass, transverse momentum and rho*calE = rho*E + rho*Phi
    (PAPER.md:14, 61-64, 210).  Insulating walls only (fixed-T walls exchange heat)."""
    if case == "periodic2d":
        prm, U = I.random_state(24, 20, 1, 7, theta=1)
        cons = [0, 1, 2, 4]
    elif case == "periodic3d":
        prm, U = I.random_state(10, 12, 9, 8, theta=1, mu=2e-3, kappa=3e-3)
        cons = [0, 1, 2, 3, 4]
    elif case == "gravity_walls2d":
        prm, U = I.random_state(16, 24, 1, 9, g=(0, -1.0, 0), bc_type=((PER, PER), (REF, REF), (0, 0)))
        cons = [0, 1, 4]
    elif case == "gravity_walls3d":
        prm, U = I.random_state(8, 10, 12, 10, g=(0, 0, -2.0), bc_type=((PER, PER), (PER, PER), (REF, REF)))
        cons = [0, 1, 2, 4]
    else:
        prm, U = I.random_state(8, 10, 12, 11, g=(0, 0, -1.0), mu=5e-3, kappa=4e-3,
                                bc_type=((PER, PER), (PER, PER), (REF, REF)))
        cons = [0, 4]          # no-stress is not imposed by a reflecting wall with viscosity: momenta may change
    shape = (prm["nz"], prm["ny"], prm["nx"])
    t0 = _totals(prm, [np.zeros(0) if a is None else a.reshape(-1) for a in
                       (U[0], U[1], U[2], U[3] if U[3] is not None else np.zeros_like(U[0]), U[4])], shape)
    S, _ = O.run(prm, U, 20, cfl=0.4)
    t1 = _totals(prm, S, shape)
    scale = [t0[0], t0[0], t0[0], t0[0], abs(t0[4])]
    for f in cons:
        assert abs(t1[f] - t0[f]) < 2e-13 * scale[f], (case, f, t0[f], t1[f])


# ----------------------------------------------------------------------------------------------- P3
def _table1():
    rows = []
    for line in open(os.path.join(GOLDEN, "table1_hydrostatic.txt")):
        if line.strip() and not line.startswith("#"):
            n, a, b = line.split()
            rows.append((int(n), float(a), float(b)))
    return rows


@pytest.mark.parametrize("theta", [0, 1])
def test_P3_isothermal_atmosphere_table1(theta):
    """PAPER.md:361-378 + Table 1: isothermal column on [0,3] initialised with (14),
    N=128, t=10.  The paper prints max|u| = 2.9e-15 (theta=1) and 1.4e-13 (theta=Ma); the values depend on
    round-off and wall closure, so the pin is the order of magnitude: within 30x of the printed number
    and far below the 1e-12 criterion of north_star."""
    n, v_theta1, v_thetaMa = _table1()[0]
    assert n == 128
    h = 3.0 / n
    T = np.ones(n)
    rho_c = I.hydrostatic_column(T, math.exp(-0.5 * h), h)
    nx = 4
    rho = np.ascontiguousarray(np.broadcast_to(rho_c[None, :, None], (1, n, nx)))
    prm = I.make_params(nx, n, 1, h, 1.4, g=(0, -1.0, 0), theta=theta,
                        bc_type=((PER, PER), (REF, REF), (0, 0)))
    U = [rho, np.zeros_like(rho), np.zeros_like(rho), None, rho / 0.4]
    # continuous solution is sampled only at the first cell; the column must follow exp(-y) to O(h^2)
    y = (np.arange(n) + 0.5) * h
    assert np.max(np.abs(rho_c - np.exp(-y)) / np.exp(-y)) < 2e-4
    t, S = 0.0, U
    while t < 10.0:
        S, dts = O.run(prm, [S[0], S[1], S[2], None, S[4]], 200, cfl=0.4)
        t += dts.sum()
        S = [S[0], S[1], S[2], None, S[4]]
    vmax = max(np.abs(S[1] / S[0]).max(), np.abs(S[2] / S[0]).max())
    ref = v_thetaMa if theta else v_theta1
    assert vmax < 30.0 * ref, (vmax, ref)
    assert vmax < 1e-12
    # density itself is unchanged to round-off
    assert np.max(np.abs(S[0] - rho.reshape(-1)) / rho.reshape(-1)) < 1e-12


def test_P3_polytrope_with_conduction_stays_at_rest():
    """Conductive polytropic layer between fixed-T no-slip walls built with (14):
    linear T => zero net conductive heating, u* = 0 => state at rest."""
    prm, U = I.config3_rb2d(nx=8, ny=48, amp=0.0)
    S, _ = O.run(prm, U, 300, cfl=0.4)
    assert max(np.abs(S[1] / S[0]).max(), np.abs(S[2] / S[0]).max()) < 1e-12
    assert np.max(np.abs(S[0] - U[0].reshape(-1))) < 1e-12
    assert np.max(np.abs(S[4] - U[4].reshape(-1)) / U[4].reshape(-1)) < 1e-12


def test_P3_sampled_exponential_is_NOT_balanced():
    """Negative control (reading A19): sampling exp(-y) at cell centres instead of (14) leaves an O(h^2)
    imbalance, i.e. the test above really exercises the discrete relation."""
    n = 64
    h = 1.0 / n
    y = (np.arange(n) + 0.5) * h
    rho = np.ascontiguousarray(np.broadcast_to(np.exp(-y)[None, :, None], (1, n, 4)))
    prm = I.make_params(4, n, 1, h, 1.4, g=(0, -1.0, 0), bc_type=((PER, PER), (REF, REF), (0, 0)))
    S, _ = O.run(prm, [rho, 0 * rho, 0 * rho, None, rho / 0.4], 100, cfl=0.4)
    assert np.abs(S[2] / S[0]).max() > 1e-9


# ----------------------------------------------------------------------------------------------- P4
@pytest.mark.parametrize("dim", [2, 3])
def test_P4_E_form_equals_calE_form(dim):
    """'both formulations are equivalent': eq. (11) on rho*calE with the relaxation Psi=Phi
    versus the rho*E + gravity-source form, on a perturbed stratified state with walls along g."""
    if dim == 2:
        prm, U = I.config1_atmosphere(32, amp=5e-2)
        U[1] = U[0] * 0.05 * np.sin(np.linspace(0, 7, U[0].size)).reshape(U[0].shape)
        U[2] = U[0] * 0.05 * np.cos(np.linspace(0, 9, U[0].size)).reshape(U[0].shape)
        U[4] = U[4] + 0.5 * (U[1] ** 2 + U[2] ** 2) / U[0]
    else:
        prm, U = I.config4_rb3d(12, amp=5e-2)
    S0, dts = O.run(prm, U, 10, cfl=0.4, form=0)
    S1, _ = O.run(prm, U, 10, dts=dts, form=1)
    for f in range(5):
        scale = np.abs(S0[f]).max() + 1e-300
        assert np.abs(S0[f] - S1[f]).max() < 2e-14 * max(scale, 1.0), f
    # negative control: the two forms are NOT trivially the same code path (energy differs from the g=0 run)
    prm0 = dict(prm, g=(0.0, 0.0, 0.0))
    Sg, _ = O.run(prm0, U, 10, dts=dts, form=0)
    assert np.abs(Sg[4] - S0[4]).max() > 1e-6


# ----------------------------------------------------------------------------------------------- P5
def _lagrange_projection_1d(rho, u, v, E, gamma, lam, K, nsteps):
    """The g=0, theta=1 scheme in the paper's OTHER formulation: Lagrangian acoustic step in specific
    variables (tau,u,v,E) with dm = rho dx, then the non-conservative transport form
    b^{n+1} = b~ - lam [b~ u*] + b~ lam [u*].  Periodic.  Independent of the oracle's
    flux form (11); pins the 1/L~ of the energy (reading A3) through rho~ = 1/tau~."""
    for _ in range(nsteps):
        e = E - 0.5 * (u * u + v * v)
        p = (gamma - 1.0) * rho * e
        c = np.sqrt(gamma * p / rho)
        rL, rR = rho, np.roll(rho, -1)
        a = K * np.maximum(rL * c, rR * np.roll(c, -1))
        us = 0.5 * (u + np.roll(u, -1)) - (np.roll(p, -1) - p) / (2 * a)        # face i+1/2
        ps = 0.5 * (p + np.roll(p, -1)) - 0.5 * a * (np.roll(u, -1) - u)
        br = lambda f: f - np.roll(f, 1)                                          # [q]_i
        tau = 1.0 / rho
        tau_t = tau + lam / rho * br(us)
        u_t = u - lam / rho * br(ps)
        v_t = v
        E_t = E - lam / rho * br(ps * us)
        rho_t = 1.0 / tau_t
        new = []
        for b in (rho_t, rho_t * u_t, rho_t * v_t, rho_t * E_t):
            bf = np.where(us >= 0, b, np.roll(b, -1))                            # upwind face value
            new.append(b - lam * br(bf * us) + b * lam * br(us))
        rho = new[0]
        u, v, E = new[1] / rho, new[2] / rho, new[3] / rho
    return rho, rho * u, rho * v, rho * E


def test_P5_reduces_to_lagrange_projection_without_gravity():
    """'in the case of a constant gravitational potential, we recover the original scheme'."""
    nx, ny = 64, 4
    x = (np.arange(nx) + 0.5) / nx
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    u = 0.4 * np.cos(2 * np.pi * x) - 0.1
    v = 0.2 * np.sin(4 * np.pi * x)
    p = 1.0 + 0.2 * np.cos(4 * np.pi * x)
    gamma = 1.4
    E = p / (gamma - 1.0) / rho + 0.5 * (u * u + v * v)
    prm = I.make_params(nx, ny, 1, 1.0 / nx, gamma, theta=0)
    bc = lambda a: np.ascontiguousarray(np.broadcast_to(a[None, None, :], (1, ny, nx)))
    U = [bc(rho), bc(rho * u), bc(rho * v), None, bc(rho * E)]
    dt = 0.2 * (1.0 / nx) / 2.0
    n = 25
    S, _ = O.run(prm, U, n, dts=np.full(n, dt))
    ref = _lagrange_projection_1d(rho, u, v, E, gamma, dt * nx, O.K(), n)
    for f, r in zip((0, 1, 2, 4), ref):
        got = S[f].reshape(ny, nx)
        assert np.abs(got - r[None, :]).max() < 1e-13, f
    # and the flow really evolved
    assert np.abs(ref[0] - rho).max() > 1e-2


# ----------------------------------------------------------------------------------------------- P6
def _exact_sod(x, t, gamma=1.4):
    """Exact Riemann solution for (1,0,1 | 0.125,0,0.1) at x0=0.5 (textbook: Newton on the pressure function)."""
    rl, pl, rr, pr = 1.0, 1.0, 0.125, 0.1
    cl, cr = math.sqrt(gamma * pl / rl), math.sqrt(gamma * pr / rr)
    g1, g2 = (gamma - 1) / (2 * gamma), (gamma + 1) / (2 * gamma)

    def f(p, rk, pk, ck):
        if p > pk:
            A, B = 2 / ((gamma + 1) * rk), (gamma - 1) / (gamma + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B))
        return 2 * ck / (gamma - 1) * ((p / pk) ** g1 - 1)

    p = 0.5 * (pl + pr)
    for _ in range(100):
        F = f(p, rl, pl, cl) + f(p, rr, pr, cr)
        dp = 1e-7 * p
        dF = (f(p + dp, rl, pl, cl) + f(p + dp, rr, pr, cr) - F) / dp
        pn = p - F / dF
        if abs(pn - p) < 1e-14:
            break
        p = pn
    ps = p
    us = 0.5 * (f(ps, rr, pr, cr) - f(ps, rl, pl, cl))
    rsl = rl * (ps / pl) ** (1 / gamma)                       # left rarefaction
    csl = cl * (ps / pl) ** g1
    rsr = rr * ((ps / pr + (gamma - 1) / (gamma + 1)) / ((gamma - 1) / (gamma + 1) * ps / pr + 1))
    S = cr * math.sqrt(g2 * ps / pr + g1)                     # shock speed
    xi = (x - 0.5) / t
    rho = np.empty_like(x)
    u = np.empty_like(x)
    pp = np.empty_like(x)
    for i, s in enumerate(xi):
        if s < -cl:
            rho[i], u[i], pp[i] = rl, 0, pl
        elif s < us - csl:
            cc = 2 / (gamma + 1) * (cl - (gamma - 1) / 2 * s)
            u[i] = 2 / (gamma + 1) * (cl + s)
            rho[i] = rl * (cc / cl) ** (2 / (gamma - 1))
            pp[i] = pl * (cc / cl) ** (2 * gamma / (gamma - 1))
        elif s < us:
            rho[i], u[i], pp[i] = rsl, us, ps
        elif s < S:
            rho[i], u[i], pp[i] = rsr, us, ps
        else:
            rho[i], u[i], pp[i] = rr, 0, pr
    return rho, u, pp, (ps, us, rsl, rsr)


def _sod_run(nx, theta):
    prm, U = I.sod_tube(nx, 4, theta=theta)
    t, S = 0.0, U
    while t < 0.2 - 1e-14:
        dt = min(O.compute_dt(prm, S, 0.4), 0.2 - t)
        S, _ = O.run(prm, S, 1, dts=[dt])
        S = [S[0], S[1], S[2], None, S[4]]
        t += dt
    rho, u, v, w, p = prim(prm, [S[0], S[1], S[2], np.zeros_like(S[0]), S[4]])
    sl = slice(0, nx)                                          # first y row
    return prm, rho[sl], u[sl], p[sl]


@pytest.mark.parametrize("theta", [0, 1])
def test_P6_sod_converges_to_exact_riemann_solution(theta):
    """correct wave speeds.  L1 errors vs the exact solution shrink under refinement and the
    star plateau approaches p*=0.30313, u*=0.92745."""
    errs = []
    for nx in (100, 200, 400):
        prm, rho, u, p = _sod_run(nx, theta)
        x = (np.arange(nx) + 0.5) / nx
        re, ue, pe, (ps, us, rsl, rsr) = _exact_sod(x, 0.2)
        errs.append((np.abs(rho - re).mean(), np.abs(u - ue).mean(), np.abs(p - pe).mean()))
        assert abs(ps - 0.30313) < 1e-5 and abs(us - 0.92745) < 1e-5 and abs(rsr - 0.26557) < 1e-5
    for q in range(3):
        assert errs[1][q] < 0.75 * errs[0][q] and errs[2][q] < 0.75 * errs[1][q], errs
    assert errs[2][0] < 1.2e-2                                  # first order, CFL 0.2 effective: diffusive but convergent
    # plateau between contact (x=0.685) and shock (x=0.850) at the finest grid
    mid = (x > 0.72) & (x < 0.82)
    assert np.abs(p[mid] - ps).max() < 0.01 and np.abs(u[mid] - us).max() < 0.02
    assert np.abs(rho[mid] - rsr).max() < 0.01
    # y-momentum stays exactly zero, solution is y-independent (transverse structure)


# ----------------------------------------------------------------------------------------------- P7
def test_P7_gresho_low_mach_correction_keeps_kinetic_energy():
    """without theta the truncation error ~ dx/Ma destroys the vortex; with eq. (13) the
    error is uniform in Ma.  64^2, Ma=1e-3, 600 steps: KE retention and L1 velocity error on vs off."""
    res = {}
    for theta in (0, 1):
        prm, U = I.config2_gresho(64, mach=1e-3, theta=theta)
        ke0 = 0.5 * ((U[1] ** 2 + U[2] ** 2) / U[0]).sum()
        S, _ = O.run(prm, U, 600, cfl=0.4)
        ke = 0.5 * ((S[1] ** 2 + S[2] ** 2) / S[0]).sum()
        l1 = (np.abs(S[1] / S[0] - (U[1] / U[0]).reshape(-1)) + np.abs(S[2] / S[0] - (U[2] / U[0]).reshape(-1))).mean()
        res[theta] = (ke / ke0, l1)
    assert res[1][0] > 0.995, res
    assert res[0][0] < 0.93, res
    assert res[0][1] > 10 * res[1][1], res
    # and at Ma=1e-1 the uncorrected scheme loses 10x less than at 1e-3 per unit of physical time ~ 1/Ma scaling
    # (same physical time: steps scale with 1/Ma)
    prm, U = I.config2_gresho(64, mach=1e-1, theta=0)
    ke0 = 0.5 * ((U[1] ** 2 + U[2] ** 2) / U[0]).sum()
    S, _ = O.run(prm, U, 6, cfl=0.4)
    loss_hi = 1 - 0.5 * ((S[1] ** 2 + S[2] ** 2) / S[0]).sum() / ke0
    assert loss_hi < (1 - res[0][0]) / 5.0, (loss_hi, res)


# ----------------------------------------------------------------------------------------------- P9
def test_P9_shear_wave_decays_by_discrete_laplacian_factor():
    """u = A sin(k y) on uniform rho, p (v=0): hyperbolic part is idle (u*_y = 0, Pi* uniform; x faces see a
    uniform-in-x state) and rho*u decays by exactly 1 - 4 (mu dt/(rho h^2)) sin^2(k h/2) in one step."""
    nx, ny = 6, 32
    h = 1.0 / ny
    mu, rho0, p0, A = 3e-3, 1.3, 2.0, 1e-2
    y = (np.arange(ny) + 0.5) * h
    kx = 2 * np.pi * 3
    u = A * np.sin(kx * y)
    full = lambda a: np.ascontiguousarray(np.broadcast_to(a[None, :, None], (1, ny, nx)))
    rho = np.full((1, ny, nx), rho0)
    U = [rho, rho * full(u), 0 * rho, None, p0 / 0.4 + 0.5 * rho * full(u) ** 2]
    prm = I.make_params(nx, ny, 1, h, 1.4, mu=mu, kappa=0.0, theta=1)
    dt = 1e-3
    S, _ = O.run(prm, U, 1, dts=[dt])
    fac = 1 - 4 * (mu * dt / (rho0 * h * h)) * math.sin(kx * h / 2) ** 2
    got = S[1].reshape(ny, nx)
    assert np.abs(got - rho0 * fac * u[:, None]).max() < 2e-16 * 10
    assert np.abs(S[0] - rho0).max() == 0.0 and np.abs(S[2]).max() < 1e-17
    # energy: total energy conserved (viscous heating moves KE -> internal only)
    assert abs(S[4].sum() - U[4].sum()) < 1e-13 * U[4].sum()
    # 3D: same wave along z carried by v; x,y uniform
    nz = 16
    hz = 1.0 / nz
    z = (np.arange(nz) + 0.5) * hz
    v = A * np.sin(2 * np.pi * 2 * z)
    full3 = lambda a: np.ascontiguousarray(np.broadcast_to(a[:, None, None], (nz, 5, 6)))
    rho3 = np.full((nz, 5, 6), rho0)
    U3 = [rho3, 0 * rho3, rho3 * full3(v), 0 * rho3, p0 / 0.4 + 0.5 * rho3 * full3(v) ** 2]
    prm3 = I.make_params(6, 5, nz, hz, 1.4, mu=mu, theta=0)
    S3, _ = O.run(prm3, U3, 1, dts=[dt])
    fac3 = 1 - 4 * (mu * dt / (rho0 * hz * hz)) * math.sin(2 * np.pi * 2 * hz / 2) ** 2
    assert np.abs(S3[2].reshape(nz, 5, 6) - rho0 * fac3 * v[:, None, None]).max() < 2e-15
    assert np.abs(S3[1]).max() < 1e-17 and np.abs(S3[3]).max() < 1e-17


def test_P9_compression_wave_sees_four_thirds_mu_and_heat_sees_kappa():
    """Linearised check of tau_dd = (2 mu - 2/3 mu) d_d u_d and of the Fourier flux:
    the DIFFERENCE between a step with (mu,kappa) and the same step with (0,0) is the parabolic operator alone
    (reading A5: evaluated on U^n, added in the same update):
      d(rho u) = dt * 4/3 mu * Lap_h u        for u = A sin(kx), v = 0
      dE       = dt * [ d_x(tau_xx ubar) + kappa Lap_h T ]."""
    nx, ny = 32, 4
    h = 1.0 / nx
    x = (np.arange(nx) + 0.5) * h
    A, k = 1e-3, 2 * np.pi * 2
    u = A * np.sin(k * x)
    T = 1.0 + 0.1 * np.cos(k * x)
    rho = np.full(nx, 1.0)
    p = rho * T
    full = lambda a: np.ascontiguousarray(np.broadcast_to(a[None, None, :], (1, ny, nx)))
    U = [full(rho), full(rho * u), full(0 * rho), None, full(p / 0.4 + 0.5 * rho * u * u)]
    mu, kappa, dt = 2e-3, 5e-3, 1e-4
    prm_v = I.make_params(nx, ny, 1, h, 1.4, mu=mu, kappa=kappa, theta=1)
    prm_0 = I.make_params(nx, ny, 1, h, 1.4, theta=1)
    Sv, _ = O.run(prm_v, U, 1, dts=[dt])
    S0, _ = O.run(prm_0, U, 1, dts=[dt])
    lap = lambda f: (np.roll(f, -1) + np.roll(f, 1) - 2 * f) / (h * h)
    dmx = (Sv[1] - S0[1]).reshape(ny, nx)[0]
    assert np.abs(dmx - dt * (4.0 / 3.0) * mu * lap(u)).max() < 1e-17
    txx = (4.0 / 3.0) * mu * (np.roll(u, -1) - u) / h                   # face i+1/2
    fe = txx * 0.5 * (u + np.roll(u, -1)) + kappa * (np.roll(T, -1) - T) / h
    dE = (Sv[4] - S0[4]).reshape(ny, nx)[0]
    assert np.abs(dE - dt * (fe - np.roll(fe, 1)) / h).max() < 1e-15
    assert np.abs(Sv[0] - S0[0]).max() == 0.0


def test_P9_cross_derivative_terms_of_the_stress_tensor():
    """tau_xy = mu (d_x v + d_y u) with the transverse derivative = mean of the two adjacent cells' centred
    differences (reading A6); eta = -2/3 mu couples d_y v into tau_xx.  A bilinear velocity
    field u = a*x*y..., whose discrete derivatives are exact, gives closed-form viscous forces on a periodic
    grid only for trigonometric fields, so use u = A sin(kx x) sin(ky y), v = B cos(kx x) cos(ky y) and the
    exact eigenvalues of the discrete operators: D0 (centred) -> i sin(kh)/h, D+- (compact) -> 2 sin(kh/2)/h."""
    n = 24
    h = 1.0 / n
    kx, ky = 2 * np.pi * 2, 2 * np.pi * 3
    xs = (np.arange(n) + 0.5) * h
    X, Y = np.meshgrid(xs, xs, indexing="xy")
    A, B, mu = 1e-3, 2e-3, 1e-2
    u = A * np.sin(kx * X) * np.sin(ky * Y)
    v = B * np.cos(kx * X) * np.cos(ky * Y)
    rho = np.ones_like(u)
    p = np.ones_like(u)
    U = [a.reshape(1, n, n) for a in (rho, rho * u, rho * v)] + [None, (p / 0.4 + 0.5 * (u * u + v * v)).reshape(1, n, n)]
    dt = 1e-4
    Sv, _ = O.run(I.make_params(n, n, 1, h, 1.4, mu=mu, theta=1), U, 1, dts=[dt])
    S0, _ = O.run(I.make_params(n, n, 1, h, 1.4, theta=1), U, 1, dts=[dt])
    lx, ly = (2 * math.sin(kx * h / 2) / h) ** 2, (2 * math.sin(ky * h / 2) / h) ** 2     # -compact Laplacian
    # mixed term: d_x(face) of [mean over the face's two cells of centred d_y]:
    #   symbol = (2 sin(kx h/2)/h) * cos(kx h/2) * (sin(ky h)/h) = sin(kx h) sin(ky h) / h^2
    mxy = math.sin(kx * h) * math.sin(ky * h) / (h * h)
    # x-momentum: d_x tau_xx + d_y tau_yx ; tau_xx = 4/3 mu u_x - 2/3 mu v_y ; tau_yx = mu (u_y + v_x)
    #   u = A sx sy, v = B cx cy:  d_x(u_x) = -lx u ; d_x(v_y): v_y = -B ky' cx sy -> d_x -> +B mxy sx sy
    fx = mu * (-(4.0 / 3.0) * lx * u - (2.0 / 3.0) * (B * mxy) * np.sin(kx * X) * np.sin(ky * Y)
               - ly * u + (B * mxy) * np.sin(kx * X) * np.sin(ky * Y))
    fy = mu * (-(4.0 / 3.0) * ly * v - (2.0 / 3.0) * (A * mxy) * np.cos(kx * X) * np.cos(ky * Y)
               - lx * v + (A * mxy) * np.cos(kx * X) * np.cos(ky * Y))
    dmx = (Sv[1] - S0[1]).reshape(n, n)
    dmy = (Sv[2] - S0[2]).reshape(n, n)
    assert np.abs(dmx - dt * fx).max() < 1e-16
    assert np.abs(dmy - dt * fy).max() < 1e-16
    assert np.abs(dt * fx).max() > 1e-9


def test_P9_rigid_translation_and_linear_T():
    """Uniform translation => zero viscous force; linear temperature between fixed-T walls => zero net heating."""
    prm, U = I.config3_rb2d(nx=8, ny=32, amp=0.0)
    prm = dict(prm, g=(0.0, 0.0, 0.0), mu=0.0)
    # uniform rho and p=rho*T linear in y would accelerate the gas; instead test the heat operator alone by
    # differencing against kappa=0 on the same (unbalanced) state
    Sk, _ = O.run(prm, U, 1, dts=[1e-5])
    S0, _ = O.run(dict(prm, kappa=0.0), U, 1, dts=[1e-5])
    # T is linear in y on the polytrope, wall ghosts continue the line (T_g = 2 T_w - T_0): zero heating
    assert np.abs(Sk[4] - S0[4]).max() < 1e-16 * np.abs(S0[4]).max() * 50
    prm2 = I.make_params(10, 12, 9, 0.1, 1.4, mu=0.05, kappa=0.0)
    shape = (9, 12, 10)
    rho = 1.0 + 0.0 * np.zeros(shape)
    U2 = [rho, 0.3 * rho, -0.2 * rho, 0.1 * rho, 2.5 + 0.5 * rho * (0.09 + 0.04 + 0.01)]
    S2, _ = O.run(prm2, U2, 3, cfl=0.4)
    for f in range(5):
        assert np.array_equal(S2[f], U2[f].reshape(-1))


# ----------------------------------------------------------------------------------------------- P10
def test_P10_axis_permutation_and_mirror_symmetry():
    """x<->y transposition in 2D, cyclic permutation in 3D, and mirror x -> -x give permuted/mirrored results."""
    prm, U = I.random_state(12, 10, 1, 21, mu=2e-3, kappa=1e-3)
    S, dts = O.run(prm, U, 5, cfl=0.4)
    Ut = [np.ascontiguousarray(np.swapaxes(a, 1, 2)) if a is not None else None for a in U]
    Ut[1], Ut[2] = Ut[2], Ut[1]
    prm_t = I.make_params(10, 12, 1, prm["dx"], prm["gamma"], mu=2e-3, kappa=1e-3)
    St, _ = O.run(prm_t, Ut, 5, dts=dts)
    back = lambda a: np.swapaxes(a.reshape(1, 12, 10), 1, 2).reshape(-1)
    for f, ft in ((0, 0), (1, 2), (2, 1), (4, 4)):
        assert np.abs(S[f] - back(St[ft])).max() < 1e-14, f
    # mirror in x: u -> -u
    Um = [np.ascontiguousarray(a[:, :, ::-1]) if a is not None else None for a in U]
    Um[1] = -Um[1]
    Sm, _ = O.run(prm, Um, 5, dts=dts)
    mir = lambda a: a.reshape(1, 10, 12)[:, :, ::-1].reshape(-1)
    for f, sgn in ((0, 1), (1, -1), (2, 1), (4, 1)):
        assert np.abs(S[f] - sgn * mir(Sm[f])).max() < 1e-14, f
    # 3D cyclic permutation (x,y,z) -> (y,z,x) with gravity along the permuted axis and walls following it
    prm3, U3 = I.random_state(6, 7, 8, 22, g=(0, 0, -1.0), mu=1e-3, kappa=2e-3,
                              bc_type=((PER, PER), (PER, PER), (FIX, REF)), bc_value=((0, 0), (0, 0), (1.7, 0)))
    S3, dts3 = O.run(prm3, U3, 4, cfl=0.4)
    # new array B[k',j',i'] with x'=z, y'=x, z'=y:  B[z'=y, y'=x, x'=z] = A[z, y, x]  -> transpose (1,2,0)
    perm = lambda a: np.ascontiguousarray(np.transpose(a, (1, 2, 0)))
    U3p = [perm(U3[0]), perm(U3[3]), perm(U3[1]), perm(U3[2]), perm(U3[4])]
    prm3p = I.make_params(8, 6, 7, prm3["dx"], prm3["gamma"], g=(-1.0, 0, 0), mu=1e-3, kappa=2e-3,
                          bc_type=((FIX, REF), (PER, PER), (PER, PER)), bc_value=((1.7, 0), (0, 0), (0, 0)))
    S3p, _ = O.run(prm3p, U3p, 4, dts=dts3)
    inv = lambda a: np.transpose(a.reshape(7, 6, 8), (2, 0, 1)).reshape(-1)
    for f, fp in ((0, 0), (1, 2), (2, 3), (3, 1), (4, 4)):
        assert np.abs(S3[f] - inv(S3p[fp])).max() < 1e-13, f


# ----------------------------------------------------------------------------------------------- ghost fill
def test_ghost_fill_periodic_and_walls():
    """Reading A9: periodic wrap == numpy 'wrap' padding; reflecting wall without gravity == mirror with the
    normal momentum negated; with gravity the ghost pair satisfies eq. (14) and T_g follows the wall kind."""
    prm, U = I.random_state(7, 6, 5, 31)
    P = O.fill_ghosts(prm, U)
    for f in range(5):
        assert np.array_equal(P[f], np.pad(U[f], 2, mode="wrap")), f
    # reflecting x walls, g = 0
    prm, U = I.random_state(7, 6, 1, 32, bc_type=((REF, REF), (PER, PER), (0, 0)))
    P = O.fill_ghosts(prm, U)
    for f, sgn in ((0, 1), (1, -1), (2, 1), (4, 1)):
        inner = np.pad(U[f], ((0, 0), (2, 2), (0, 0)), mode="wrap")        # y periodic
        assert np.allclose(P[f][:, :, 1], sgn * inner[:, :, 0], rtol=3e-16 * 8, atol=0), f     # ghost -1 <- cell 0
        assert np.allclose(P[f][:, :, -2], sgn * inner[:, :, -1], rtol=3e-16 * 8, atol=0), f
    # layer 2 takes velocity and temperature of interior cell 1 and chains eq. (14) from layer 1: with g = 0
    # that means p_g2 = p_g1 (= p of cell 0), T_g2 = T_1, u_g2 = -u_1, v_g2 = v_1
    gm1 = prm["gamma"] - 1
    pr = lambda A, i: gm1 * (A[4][:, :, i] - 0.5 * (A[1][:, :, i] ** 2 + A[2][:, :, i] ** 2) / A[0][:, :, i])
    for g2, g1, c1 in ((0, 1, 3), (-1, -2, -4)):
        assert np.allclose(pr(P, g2), pr(P, g1), rtol=1e-14, atol=0)
        assert np.allclose(pr(P, g2) / P[0][:, :, g2], pr(P, c1) / P[0][:, :, c1], rtol=1e-14, atol=0)
        assert np.allclose(P[1][:, :, g2] / P[0][:, :, g2], -P[1][:, :, c1] / P[0][:, :, c1], rtol=1e-14, atol=0)
        assert np.allclose(P[2][:, :, g2] / P[0][:, :, g2], P[2][:, :, c1] / P[0][:, :, c1], rtol=1e-14, atol=0)
    # gravity + fixed-T bottom, reflecting top, 3D, z walls
    Tw = 1.9
    prm, U = I.random_state(5, 6, 7, 33, g=(0, 0, -1.5), bc_type=((PER, PER), (PER, PER), (FIX, REF)),
                            bc_value=((0, 0), (0, 0), (Tw, 0)), h=0.05)
    P = O.fill_ghosts(prm, U)
    gm1 = prm["gamma"] - 1
    rho, mx, my, mz, E = P
    p = gm1 * (E - 0.5 * (mx ** 2 + my ** 2 + mz ** 2) / rho)
    T = p / rho
    dphi = 1.5 * 0.05                                                      # Phi_{k+1} - Phi_k
    for k in (0, 1, 7 + 2, 7 + 3 - 1 + 0):                                 # pairs (k,k+1) that involve a ghost
        lhs = p[k + 1] - p[k]
        rhs = -0.5 * (rho[k] + rho[k + 1]) * dphi
        assert np.abs(lhs - rhs).max() < 1e-14, k
    assert np.abs(0.5 * (T[1] + T[2]) - Tw).max() < 1e-14                  # wall-face temperature
    assert np.abs(0.5 * (T[0] + T[3]) - Tw).max() < 1e-14
    for m in (mx, my, mz):                                                 # no-slip: all components flip
        assert np.abs(m[1] / rho[1] + m[2] / rho[2]).max() < 1e-15
    assert np.abs(T[-2] - T[-3]).max() < 1e-14                             # insulating top: T copied
    assert np.abs(mz[-2] / rho[-2] + mz[-3] / rho[-3]).max() < 1e-15       # normal flips
    assert np.abs(mx[-2] / rho[-2] - mx[-3] / rho[-3]).max() < 1e-15       # tangential copied
    # corners are filled (finite, positive density) -- needed by the diagonal viscous stencil
    assert np.all(np.isfinite(rho)) and rho.min() > 0


# ----------------------------------------------------------------------------------------------- CFL
def test_cfl_closed_form_and_stability_margin():
    """Reading A4.  Uniform state: closed form.  And the property the formula exists for: with cfl=0.4 the
    acoustic Jacobian L~ = 1 + lam sum[u*] stays positive and the update keeps rho, p > 0 on a violent state."""
    prm = I.make_params(6, 5, 4, 0.02, 1.4, mu=1e-3, kappa=4e-3)
    rho, u, v, w, p = 0.8, 0.3, -0.6, 0.2, 1.7
    shape = (4, 5, 6)
    E = p / 0.4 + 0.5 * rho * (u * u + v * v + w * w)
    U = [np.full(shape, x) for x in (rho, rho * u, rho * v, rho * w, E)]
    c = math.sqrt(1.4 * p / rho)
    r = (abs(u) + abs(v) + abs(w) + 3 * c) / 0.02 + 2 * 3 * max(4e-3 / 3, 0.4 * 4e-3) / (rho * 0.02 ** 2)
    assert abs(O.max_rate(prm, U) - r) < 1e-12 * r
    prm2 = dict(prm, nz=1, ny=5, nx=24, mu=0.0, kappa=0.0)
    U2 = [np.full((1, 5, 24), x) for x in (rho, rho * u, rho * v)] + [None, np.full((1, 5, 24), p / 0.4 + 0.5 * rho * (u * u + v * v))]
    r2 = (abs(u) + abs(v) + 2 * c) / 0.02
    assert abs(O.max_rate(prm2, U2) - r2) < 1e-12 * r2
    # the max picks the single fastest cell
    U2[1][0, 3, 17] = rho * 5.0
    U2[4][0, 3, 17] += 0.5 * rho * (25.0 - u * u)
    assert abs(O.max_rate(prm2, U2) - (5.0 + abs(v) + 2 * c) / 0.02) < 1e-10
    # NaN / negative pressure is reported, not hidden
    U2[4][0, 0, 0] = -1.0
    assert math.isnan(O.max_rate(prm2, U2))
    with pytest.raises(FloatingPointError):
        O.run(prm2, U2, 1, cfl=0.4)
    # strong 2D blast: positivity over 60 steps at cfl 0.4
    prm3, U3 = I.random_state(32, 32, 1, 5, vel=0.0)
    U3[4][0, 12:20, 12:20] *= 50.0
    S, _ = O.run(prm3, U3, 60, cfl=0.4)
    rho_, u_, v_, w_, p_ = prim(prm3, S)
    assert rho_.min() > 0 and p_.min() > 0


# ----------------------------------------------------------------------------------------------- imposed-flux wall (A22)
FLX = I.BC_FLUX


def test_flux_wall_energy_budget_closed_form():
    """PAPER.md:435 "we impose the temperature flux on the bottom boundary" (reading A22).  With u*_wall = 0 the only
    energy that crosses a flux wall is the conductive flux kappa (T_ghost - T_0)/h = F, so per step
    Delta sum(E + rho Phi) = dt * (face cells) * (F_lo + F_hi) / h exactly, and mass is conserved (mu = 0: no wall stress
    work; the state is a random one, not an equilibrium)."""
    for dim in (2, 3):
        Flo, Fhi = 0.037, -0.011
        if dim == 2:
            prm, U = I.random_state(12, 16, 1, 21, g=(0, -1.0, 0), mu=0.0, kappa=5e-2,
                                    bc_type=((PER, PER), (FLX, FLX), (0, 0)), bc_value=((0, 0), (Flo, Fhi), (0, 0)))
            nface = prm["nx"]
        else:
            prm, U = I.random_state(6, 7, 10, 22, g=(0, 0, -1.0), mu=0.0, kappa=5e-2,
                                    bc_type=((PER, PER), (PER, PER), (FLX, FLX)), bc_value=((0, 0), (0, 0), (Flo, Fhi)))
            nface = prm["nx"] * prm["ny"]
        shape = (prm["nz"], prm["ny"], prm["nx"])
        S = [a if a is not None else np.zeros_like(U[0]) for a in U]
        for _ in range(5):
            t0 = _totals(prm, [a.reshape(-1) for a in S], shape)
            S, dts = O.run(prm, S, 1, cfl=0.4)
            t1 = _totals(prm, S, shape)
            expect = dts[0] * nface * (Flo + Fhi) / prm["dx"]
            assert abs((t1[4] - t0[4]) - expect) < 1e-12 * abs(t0[4]), (dim, t1[4] - t0[4], expect)
            assert abs(t1[0] - t0[0]) < 1e-13 * t0[0]


def test_flux_wall_with_zero_flux_is_the_reflecting_wall():
    prm, U = I.random_state(14, 12, 1, 23, g=(0, -1.0, 0), mu=1e-3, kappa=2e-3, bc_type=((PER, PER), (FLX, FLX), (0, 0)))
    ref = dict(prm, bc_type=((PER, PER), (REF, REF), (0, 0)))
    A, _ = O.run(prm, U, 4, cfl=0.4)
    B, _ = O.run(ref, U, 4, cfl=0.4)
    for f in (0, 1, 2, 4):
        assert np.array_equal(A[f], B[f]), f


def test_flux_wall_feeding_the_conductive_flux_keeps_the_polytrope_at_rest():
    """The paper's 2D Rayleigh-Benard walls: temperature flux imposed at the bottom, here equal to the
    conductive flux kappa*beta of the linear profile, fixed temperature at the top: the layer built with (14) is a
    steady state of the scheme (the wall face carries exactly the flux every interior face carries)."""
    prm, U = I.config3_rb2d(nx=8, ny=48, amp=0.0)
    beta = 1.0 / 2.3
    bt = ((PER, PER), (FLX, FIX), (0, 0))
    bv = ((0, 0), (prm["kappa"] * beta, prm["bc_value"][1][1]), (0, 0))
    prm = dict(prm, bc_type=bt, bc_value=bv)
    S, _ = O.run(prm, U, 300, cfl=0.4)
    # a flux wall reflects the velocity (free slip): the rest state must survive it as it does the no-slip wall
    assert max(np.abs(S[1] / S[0]).max(), np.abs(S[2] / S[0]).max()) < 1e-12
    assert np.max(np.abs(S[4] - U[4].reshape(-1)) / U[4].reshape(-1)) < 1e-12


# ----------------------------------------------------------------------------------------------- diagnostics
def test_diagnostics_closed_forms():
    """PAPER.md:398-407 (maximum velocity), :435 (mean absolute velocity), :14 (mass, total energy).  Uniform state under
    gravity: every entry has a closed form (sum of cell-centre heights = n L / 2); a single fast cell moves the two
    maxima and nothing else by more than its own share."""
    nx, ny, nz, h, gamma = 6, 5, 4, 0.25, 1.4
    rho, u, v, w, p = 1.25, 0.3, -0.4, 1.2, 0.75
    g = (0.0, 0.5, -2.0)
    prm = I.make_params(nx, ny, nz, h, gamma, g=g)
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)
    U = [np.full((nz, ny, nx), x) for x in (rho, rho * u, rho * v, rho * w, E)]
    d = O.diagnostics(prm, U)
    speed = math.sqrt(u * u + v * v + w * w)          # = 1.3
    V = nx * ny * nz * h ** 3
    assert abs(d["max_speed"] - speed) < 1e-15 and abs(d["mean_speed"] - speed) < 1e-15
    assert abs(d["kinetic_energy"] - 0.5 * rho * speed ** 2 * V) < 1e-13
    assert abs(d["max_mach"] - speed / math.sqrt(gamma * p / rho)) < 1e-15
    assert abs(d["mass"] - rho * V) < 1e-13
    # Phi = -g.x: mean height of the cell centres along an axis of n cells is n h / 2
    phi_mean = -(g[1] * ny * h / 2 + g[2] * nz * h / 2)
    assert abs(d["total_energy"] - (E + rho * phi_mean) * V) < 1e-12
    s2 = math.sqrt(u * u + v * v + 25.0)
    U[3][2, 1, 3] = rho * 5.0                          # one fast cell at the same pressure
    U[4][2, 1, 3] = p / (gamma - 1) + 0.5 * rho * s2 * s2
    d2 = O.diagnostics(prm, U)
    assert abs(d2["max_speed"] - s2) < 1e-14
    assert abs(d2["mean_speed"] - (speed * (nx * ny * nz - 1) + s2) / (nx * ny * nz)) < 1e-14
    assert abs(d2["max_mach"] - s2 / math.sqrt(gamma * p / rho)) < 1e-13 and abs(d2["mass"] - d["mass"]) < 1e-13


def test_wall_closure_needs_a_positive_ghost_density():
    """Reading A9: relation (14) gives rho_g = (p + rho delta / 2) / (T_g - delta / 2), which is only a
    density when T_g > |g| h / 2.  Closed form on one column: with T_g below that bound the ghost cell is flagged
    (NaN) and max_rate of the ghost-filled state is non-finite; just above it the ghost density is positive and obeys
    relation (14) exactly."""
    for T, ok in ((0.6, True), (0.4, False)):
        prm = I.make_params(4, 4, 1, 1.0, 1.4, g=(0.0, -1.0, 0.0), bc_type=((PER, PER), (REF, REF), (0, 0)))
        rho = np.full((1, 4, 4), 2.0)
        p = rho * T
        U = [rho, np.zeros_like(rho), np.zeros_like(rho), None, p / 0.4]
        G = O.fill_ghosts(prm, U)
        top = G[0][0, -2, 2:-2]                 # first ghost layer above the top wall: delta = Phi_prev - Phi_g = -|g| h
        bot = G[0][0, 1, 2:-2]                  # first ghost layer below the bottom wall: delta = +|g| h
        if ok:
            assert np.allclose(top, (2.0 * T - 0.5 * 2.0) / (T + 0.5), rtol=1e-15) and (top > 0).all()
            assert np.allclose(bot, (2.0 * T + 0.5 * 2.0) / (T - 0.5), rtol=1e-14) and (bot > 0).all()
        else:
            assert np.isnan(top).all() and np.isnan(bot).all()


def test_rayleigh_taylor_equilibrium_is_preserved_without_perturbation():
    """'We do not need to use the well-balanced formula (14), the equilibrium is preserved in the case
    A = 0': the two-layer Rayleigh-Taylor state (rho = 1 | 2, p linear in y on each side, reading A23) satisfies the
    discrete balance (14) exactly, interface face included, so it stays at rest to round-off with and without the
    low-Mach correction; with the C = 0.01 perturbation the heavy fluid starts to fall (kinetic energy grows)."""
    for theta in (1, 0):
        prm, U = I.rayleigh_taylor(16, 48, C=0.0, theta=theta)
        S, _ = O.run(prm, U, 400, cfl=0.4)
        assert np.abs(S[2] / S[0]).max() < 1e-13 and np.abs(S[1]).max() == 0.0
        assert abs(S[0].sum() - U[0].sum()) <= 1e-13 * U[0].sum()
    # the seeded mode grows exponentially (PAPER.md:421 'we recover the classical linear growing mode'): after the
    # acoustic transient the kinetic energy multiplies by > 2.5 per 500 steps (t ~ 1.65), at a rate below the sharp-
    # interface inviscid value 2 sqrt(A g k) = 1.29 (A = 1/3, g = 0.1, k = 4 pi)
    prm, U = I.rayleigh_taylor(16, 48)
    S, ke, t = U, [], []
    for _ in range(4):
        S, dts = O.run(prm, S, 500, cfl=0.4)
        ke.append((0.5 * (S[1] ** 2 + S[2] ** 2) / S[0]).sum())
        t.append(dts.sum())
        S = [S[0], S[1], S[2], None, S[4]]
    for a, b, dt in zip(ke[:-1], ke[1:], t[1:]):
        assert 2.5 < b / a < np.exp(1.29 * dt)


def test_strongly_stratified_polytrope_with_flux_bottom_is_steady():
    """the chi = 21 polytrope initialised by recursion (14), heated from below by exactly its own
    conductive flux (imposed-flux wall, reading A22) and held at T_top above, is a steady state: it stays at rest."""
    prm, U = I.rb2d_chi21(24, 32, amp=0.0)
    assert 15.0 < U[0].max() / U[0].min() < 21.0          # cell-centre density contrast of the chi = 21 layer
    S, _ = O.run(prm, U, 500, cfl=0.4)
    assert np.abs(S[2] / S[0]).max() < 1e-12
    E0 = U[4].sum()
    assert abs(S[4].sum() - E0) < 1e-12 * E0              # heat in at the bottom = heat out at the top


# ----------------------------------------------------------------------------------- Appendix B, general potential
def _appendix_b_lagrangian_1d(rho, u, v, E, Phi, gamma, lam, K, nsteps):
    """The non-conservative scheme of Appendix B in the paper's OTHER formulation: the Lagrangian
    acoustic system in (tau, u, v, E) with its sources -(1/tau) d_m Phi and -(u/tau) d_m Phi, dm = rho dx, face source
    S_{i+1/2} = -1/2 (1/tau_i + 1/tau_{i+1}) (Phi_{i+1} - Phi_i), then the non-conservative transport
    form b^{n+1} = b~ - lam [b~ u*] + b~ lam [u*].  Periodic, theta = 1.  Independent of the oracle's flux form."""
    for _ in range(nsteps):
        e = E - 0.5 * (u * u + v * v)
        p = (gamma - 1.0) * rho * e
        c = np.sqrt(gamma * p / rho)
        up = lambda f: np.roll(f, -1)
        a = K * np.maximum(rho * c, up(rho) * up(c))
        S = -0.5 * (rho + up(rho)) * (up(Phi) - Phi)                                 # face i+1/2
        us = 0.5 * (u + up(u)) - (up(p) - p - S) / (2 * a)
        ps = 0.5 * (p + up(p)) - 0.5 * a * (up(u) - u)
        br = lambda f: f - np.roll(f, 1)                                            # [q]_i
        Si = 0.5 * (S + np.roll(S, 1))
        uSi = 0.5 * (us * S + np.roll(us * S, 1))
        tau_t = 1.0 / rho + lam / rho * br(us)
        u_t = u - lam / rho * br(ps) + lam / rho * Si
        E_t = E - lam / rho * br(ps * us) + lam / rho * uSi
        rho_t = 1.0 / tau_t
        new = []
        for b in (rho_t, rho_t * u_t, rho_t * v, rho_t * E_t):
            bf = np.where(us >= 0, b, up(b))
            new.append(b - lam * br(bf * us) + b * lam * br(us))
        rho = new[0]
        u, v, E = new[1] / rho, new[2] / rho, new[3] / rho
    return rho, rho * u, rho * v, rho * E


def _wave_1d(nx, ny):
    x = (np.arange(nx) + 0.5) / nx
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    u = 0.4 * np.cos(2 * np.pi * x) - 0.1
    v = 0.2 * np.sin(4 * np.pi * x)
    p = 1.0 + 0.2 * np.cos(4 * np.pi * x)
    E = p / 0.4 / rho + 0.5 * (u * u + v * v)
    bc = lambda a: np.ascontiguousarray(np.broadcast_to(a[None, None, :], (1, ny, nx)))
    return x, (rho, u, v, E), [bc(rho), bc(rho * u), bc(rho * v), None, bc(rho * E)], bc


def test_appendix_B_scheme_matches_its_lagrangian_formulation_with_a_general_potential():
    """Oracle form 2 (App. B, reading A24) with an array-valued periodic potential
    against an independent implementation of the Lagrangian formulation the appendix starts from."""
    nx, ny = 64, 4
    x, (rho, u, v, E), U, bc = _wave_1d(nx, ny)
    Phi = 0.3 * np.sin(2 * np.pi * x) + 0.1 * np.cos(6 * np.pi * x)
    prm = dict(I.make_params(nx, ny, 1, 1.0 / nx, 1.4, theta=0), phi=bc(Phi))
    dt = 0.2 * (1.0 / nx) / 2.0
    n = 25
    S, _ = O.run(prm, U, n, dts=np.full(n, dt), form=2)
    ref = _appendix_b_lagrangian_1d(rho, u, v, E, Phi, 1.4, dt * nx, O.K(), n)
    for f, r in zip((0, 1, 2, 4), ref):
        assert np.abs(S[f].reshape(ny, nx) - r[None, :]).max() < 1e-13, f
    # the potential really acted, and the energy form matters: form 0 gives another energy, the same mass
    S0, _ = O.run(dict(prm, phi=None), U, n, dts=np.full(n, dt), form=2)
    assert np.abs(S0[1] - S[1]).max() > 1e-3
    Sc, _ = O.run(prm, U, n, dts=np.full(n, dt), form=0)
    assert np.abs(Sc[4] - S[4]).max() > 1e-7 and np.abs(Sc[4] - S[4]).max() < 1e-2


def test_appendix_B_coincides_with_the_conservative_scheme_where_it_must():
    """Without gravity the two energy updates are the same expression (S = 0): bit-identical.  At rest in a
    hydrostatic column u* = 0 on every face, so (uS)_i = 0 and the well-balanced property carries
    over: the isothermal atmosphere stays at rest.  With gravity and flow the total energy sum(E + rho Phi) is conserved
    to round-off by the conservative forms only."""
    prm, U = I.random_state(18, 14, 6, 41, mu=1e-3, kappa=2e-3)
    A, _ = O.run(prm, U, 4, cfl=0.4, form=0)
    B, _ = O.run(prm, U, 4, cfl=0.4, form=2)
    for f in range(5):
        assert np.array_equal(A[f], B[f]), f
    prm, U = I.config1_atmosphere(32, amp=0.0)
    S, _ = O.run(prm, U, 300, cfl=0.4, form=2)
    assert np.abs(S[2] / S[0]).max() < 1e-13
    prm, U = I.config1_atmosphere(32, amp=1e-2)
    y = (np.arange(32) + 0.5) / 32
    tot = lambda S: (S[4].reshape(32, 32) + S[0].reshape(32, 32) * y[:, None]).sum()
    e0 = (U[4][0] + U[0][0] * y[:, None]).sum()
    A, _ = O.run(prm, U, 50, cfl=0.4, form=0)
    B, _ = O.run(prm, U, 50, cfl=0.4, form=2)
    assert abs(tot(A) - e0) < 1e-12 * e0
    assert 1e-12 * e0 < abs(tot(B) - e0) < 1e-5 * e0
    assert abs(B[0].sum() - U[0].sum()) < 1e-13 * U[0].sum()


def test_array_potential_reduces_to_constant_gravity_and_keeps_the_two_energy_forms_equivalent():
    """S_{i+1/2} = -1/2 (rho_i + rho_{i+1}) (Phi_{i+1} - Phi_i).  (a) Phi = -g.x sampled at the cell
    centres (values exactly representable: h = 1/16, g = (0.5, -1, 0.25)) reproduces the constant-g run: the face sources
    are bit-identical, the gravity work differs only by the rounding of lam (g h) m against dt g m.  (b) With a smooth
    non-linear potential the rho E + source form and the calligraphic-E form (11) still agree to round-off,
    which pins the upwind-potential gravity work.  (c) A column in discrete hydrostatic balance (14) with that potential
    stays at rest."""
    PERp, REFp = I.BC_PERIODIC, I.BC_REFLECTING
    n = 16
    h = 1.0 / n
    g = (0.5, -1.0, 0.25)
    prm, U = I.random_state(n, n, n, 43, g=g, h=h, mu=1e-3, kappa=1e-3,
                            bc_type=((REFp, REFp), (REFp, I.BC_FIXED_T), (REFp, REFp)), bc_value=((0, 0), (0, 2.5), (0, 0)))
    c = (np.arange(n) + 0.5) * h
    Phi = -(g[0] * c[None, None, :] + g[1] * c[None, :, None] + g[2] * c[:, None, None])
    A, dts = O.run(prm, U, 5, cfl=0.4)
    B, _ = O.run(dict(prm, phi=Phi), U, 5, dts=dts)
    for f in range(4):
        assert np.array_equal(A[f], B[f]) or np.abs(A[f] - B[f]).max() < 2e-15 * np.abs(A[f]).max(), f
    assert np.abs(A[4] - B[4]).max() < 1e-14 * np.abs(A[4]).max()
    # (b) non-linear potential, periodic in x and y, walls in z
    prm, U = I.random_state(12, 10, 8, 44, bc_type=((PERp, PERp), (PERp, PERp), (REFp, REFp)), h=1.0 / 12)
    x = (np.arange(12) + 0.5) / 12
    yy = (np.arange(10) + 0.5) / 10
    z = (np.arange(8) + 0.5) / 12
    Phi = 0.2 * np.sin(2 * np.pi * x)[None, None, :] * np.cos(2 * np.pi * yy)[None, :, None] + (0.8 * z + 0.5 * z * z)[:, None, None]
    pp = dict(prm, phi=Phi)
    A, dts = O.run(pp, U, 6, cfl=0.3, form=0)
    B, _ = O.run(pp, U, 6, dts=dts, form=1)
    for f in range(5):
        assert np.abs(A[f] - B[f]).max() < 5e-14 * np.abs(A[f]).max(), f
    etot = lambda S: (S[4] + S[0] * Phi.reshape(-1)).sum()
    e0 = (U[4] + U[0] * Phi).sum()
    assert abs(etot(A) - e0) < 1e-13 * abs(e0)                 # sum (E + rho Phi) is conserved
    assert np.abs(A[3] - O.run(prm, U, 6, dts=dts)[0][3]).max() > 1e-3   # and the potential really acted
    # (c) hydrostatic column in a non-uniform field g(y) = 1 + y: Phi = y + y^2 / 2, T = 1, recursion (14) with the local dPhi
    ny = 48
    hy = 1.0 / ny
    yc = (np.arange(ny) + 0.5) * hy
    Phic = yc + 0.5 * yc * yc
    rho = np.empty(ny)
    rho[0] = 1.0
    for j in range(ny - 1):
        d = Phic[j + 1] - Phic[j]
        rho[j + 1] = rho[j] * (1.0 - 0.5 * d) / (1.0 + 0.5 * d)
    prmc = I.make_params(8, ny, 1, hy, 1.4, bc_type=((PERp, PERp), (REFp, REFp), (0, 0)))
    col = lambda a: np.ascontiguousarray(np.broadcast_to(a[None, :, None], (1, ny, 8)))
    Uc = [col(rho), col(0 * rho), col(0 * rho), None, col(rho / 0.4)]
    S, _ = O.run(dict(prmc, phi=col(Phic)), Uc, 400, cfl=0.4)
    assert np.abs(S[2] / S[0]).max() < 1e-13


# ---------------------------------------------------------------------------------------------------------------
# mid-plane kinetic-energy spectrum (reading A26)
# ---------------------------------------------------------------------------------------------------------------
def test_ke_spectrum_parseval_single_mode_and_brute_force():
    rng = np.random.default_rng(5)
    nx, ny, nz = 12, 10, 8
    prm = I.make_params(nx, ny, nz, 0.1, 1.4)
    rho = 0.5 + rng.random((nz, ny, nx))
    vel = [rng.standard_normal((nz, ny, nx)) for _ in range(3)]
    U = [rho, rho * vel[0], rho * vel[1], rho * vel[2], np.ones((nz, ny, nx))]
    E = O.ke_spectrum(prm, U)
    k = nz // 2
    # Parseval: the shells add up to the plane mean of 1/2 rho |u|^2
    mean_ke = float((0.5 * rho[k] * (vel[0][k] ** 2 + vel[1][k] ** 2 + vel[2][k] ** 2)).mean())
    assert abs(E.sum() - mean_ke) < 1e-13 * mean_ke
    assert E.size == int(np.floor(np.hypot(nx // 2, ny // 2) + 0.5)) + 1
    # brute force: the double sum of the definition, term by term
    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    brute = np.zeros(E.size)
    for qy in range(ny):
        for qx in range(nx):
            ph = np.exp(-2j * np.pi * (qx * i / nx + qy * j / ny))
            pw = sum(0.5 * abs((np.sqrt(rho[k]) * vel[c][k] * ph).sum() / (nx * ny)) ** 2 for c in range(3))
            sx, sy = (qx if 2 * qx <= nx else qx - nx), (qy if 2 * qy <= ny else qy - ny)
            brute[int(np.floor(np.hypot(sx, sy) + 0.5))] += pw
    assert np.abs(E - brute).max() < 1e-13 * brute.max()
    # one Fourier mode u = a cos(2 pi (3 i / nx + 2 j / ny)), rho = 1: |w^| = a/2 at +-(3,2), shell round(sqrt(13)) = 4, E = a^2/4
    a = 0.7
    u = a * np.cos(2 * np.pi * (3 * i / nx + 2 * j / ny))
    one = np.ones((nz, ny, nx))
    E1 = O.ke_spectrum(prm, [one, one * u[None], 0 * one, 0 * one, one])
    expect = np.zeros(E.size); expect[4] = a * a / 4
    assert np.abs(E1 - expect).max() < 1e-15


def test_oracle_is_clean_under_asan_ubsan(tmp_path):
    """SURVEY section 5 (sanitizer row): oracle/ark_oracle.cpp built into a stand-alone executable with
    -fsanitize=address,undefined and run on small 2D / 3D cases with every wall kind, the three energy forms and an
    array-valued potential (tests/oracle_sanitizer_main.cpp).  Any out-of-bounds access, use of an uninitialised vector
    slot beyond its size, signed overflow or misaligned access aborts the run (-fno-sanitize-recover)."""
    import shutil
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    exe = str(tmp_path / "oracle_asan")
    cmd = ["g++", "-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-o", exe, os.path.join(root, "tests", "oracle_sanitizer_main.cpp"), os.path.join(root, "oracle", "ark_oracle.cpp")]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and ("asan" in b.stderr or "ubsan" in b.stderr or "sanitize" in b.stderr):
        pytest.skip("sanitizer runtime not installed: " + b.stderr.strip().splitlines()[-1])
    assert b.returncode == 0, b.stderr
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1"))
    assert r.returncode == 0, (r.stdout, r.stderr)
    assert r.stdout.count(" ok ") == 5 and "ERROR" not in r.stderr and "runtime error" not in r.stderr, (r.stdout, r.stderr)
