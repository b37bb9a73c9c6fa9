"""CPU check of the CUDA kernel SOURCES: paper_1903_09043_b200/csrc/*.cuh compiled with g++ under the test-only
host emulation shim (tests/emu/ark_emu.h: one std::thread per CUDA thread, __syncthreads = barrier) and compared
with the oracle.  Exercises tiling, halo, ragged tiles, z chunks, the register/shared-memory pipeline, the ghost
fill and both CFL paths.  The emulated build is not the product (that is nvcc-built libark_b200.so, tested by the
`-m gpu` parity tests)."""
import numpy as np
import pytest

from oracle import ark_oracle as O
from paper_1903_09043_b200 import inputs as I
from tests.emu import emu

PER, REF, FIX = I.BC_PERIODIC, I.BC_REFLECTING, I.BC_FIXED_T


def _compare(prm, U, nsteps, zchunk=0, tol=5e-14):
    S0, dts = O.run(prm, U, nsteps, cfl=0.4)
    S1, rates, rate0 = emu.run(prm, U, dts, zchunk)
    for f in range(5):
        scale = np.abs(S0[f]).max()
        assert np.abs(S0[f] - S1[f]).max() <= tol * max(scale, 1e-300), (f, np.abs(S0[f] - S1[f]).max(), scale)
    r0 = O.max_rate(prm, U)
    assert abs(rate0 - r0) <= 1e-14 * r0                                  # standalone two-pass reduction
    rN = O.max_rate(prm, [S0[0], S0[1], S0[2], S0[3], S0[4]])
    assert abs(rates[-1] - rN) <= 1e-12 * rN                              # fused epilogue + pass 2


CASES = {
    "2d_periodic_inviscid": lambda: I.random_state(20, 10, 1, 3),
    "2d_theta_off": lambda: I.random_state(17, 9, 1, 13, theta=0),
    "2d_walls_gravity_viscous": lambda: I.random_state(19, 11, 1, 4, mu=2e-3, kappa=3e-3, g=(0, -1.0, 0),
                                                       bc_type=((PER, PER), (FIX, REF), (0, 0)),
                                                       bc_value=((0, 0), (1.5, 0), (0, 0))),
    "2d_gravity_x_walls_x": lambda: I.random_state(13, 8, 1, 14, g=(-0.7, 0.3, 0),
                                                   bc_type=((REF, REF), (REF, REF), (0, 0))),
    "2d_flux_wall": lambda: I.random_state(15, 10, 1, 24, mu=1e-3, kappa=5e-2, g=(0, -1.0, 0),
                                           bc_type=((PER, PER), (I.BC_FLUX, FIX), (0, 0)), bc_value=((0, 0), (0.03, 1.5), (0, 0))),
    "3d_flux_wall": lambda: I.random_state(9, 8, 9, 25, mu=1e-3, kappa=5e-2, g=(0, 0, -1.0),
                                           bc_type=((PER, PER), (PER, PER), (I.BC_FLUX, REF)), bc_value=((0, 0), (0, 0), (0.03, 0))),
    "3d_periodic_inviscid": lambda: I.random_state(12, 9, 7, 5),
    "3d_walls_gravity_viscous": lambda: I.random_state(12, 9, 10, 6, mu=2e-3, kappa=3e-3, g=(0, 0, -1.0),
                                                       bc_type=((PER, PER), (PER, PER), (FIX, REF)),
                                                       bc_value=((0, 0), (0, 0), (1.5, 0))),
    "3d_all_walls_oblique_gravity": lambda: I.random_state(9, 10, 8, 7, mu=1e-3, kappa=0.0, g=(0.2, -0.3, -1.0),
                                                           bc_type=((REF, FIX), (FIX, REF), (REF, REF)),
                                                           bc_value=((0, 2.5), (2.2, 0), (0, 0))),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_emulated_kernels_match_oracle(name):
    prm, U = CASES[name]()
    _compare(prm, U, 3)


def test_emulated_z_chunks_and_prologue():
    prm, U = CASES["3d_walls_gravity_viscous"]()
    _compare(prm, U, 2, zchunk=4)      # 10 planes -> chunks of 4,4,2
    _compare(prm, U, 2, zchunk=3)


def test_emulated_config_shapes():
    # momenta of the perturbed atmospheres are ~1e-5 while their round-off floor is set by O(1) pressure terms
    # (reading A20): use north_star's 1e-11 here, the 5e-14 of the O(1) random states above would be too tight
    # (config 5's chi = 100 polytrope needs >= 50 cells per height for a positive ghost density at the top wall, reading
    # A9; the 8^3 stand-in keeps its recipe -- imposed-flux bottom, reflecting top, velocity noise -- with chi = 3)
    c5 = I._convection3d(8, 8, 1.0, 3.0, 1.0e-4, 2.5e-4, I.BC_REFLECTING, 1e-2, 1005, 1, None, None, heat=10.0)
    for prm, U in (I.config1_atmosphere(12), I.config3_rb2d(12, 8), I.config4_rb3d(8), c5):
        _compare(prm, U, 3, tol=1e-11)


def test_emulated_ghost_fill_matches_oracle():
    for name in ("2d_walls_gravity_viscous", "3d_all_walls_oblique_gravity", "3d_periodic_inviscid"):
        prm, U = CASES[name]()
        ref = O.fill_ghosts(prm, U)
        _, _, _, padded = emu.run(prm, U, [1e-6], want_padded=True)
        fields = [0, 1, 2, 3, 4] if prm["nz"] > 1 else [0, 1, 2, 4]
        for slot, f in enumerate(fields):
            a, b = padded[slot], ref[f]
            assert np.abs(a - b).max() <= 4e-15 * np.abs(b).max(), (name, f)


def test_emulated_nan_propagates_to_rate():
    prm, U = I.random_state(12, 8, 1, 9)
    U[4][0, 3, 5] = -5.0                       # negative pressure -> NaN sound speed
    _, _, rate0 = emu.run(prm, U, [])
    assert np.isnan(rate0)


def _phi_field(nx, ny, nz, h, kind):
    """A smooth non-linear potential at the cell centres (dense, x fastest)."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    x, y, z = (i + 0.5) * h, (j + 0.5) * h, (k + 0.5) * h
    if kind == "periodic":
        return 0.3 * np.cos(2 * np.pi * x / (nx * h)) * np.cos(2 * np.pi * y / (ny * h)) * (np.cos(2 * np.pi * z / (nz * h)) if nz > 1 else 1.0)
    return 0.8 * y + 0.5 * y * y + 0.2 * np.sin(2 * np.pi * x / (nx * h)) + (0.6 * z + 0.3 * z * z * y if nz > 1 else 0.0)


GEN_CASES = {
    # SURVEY 8(f) row 4 (Appendix B) and row 2 (array-valued potential)
    "2d_appendix_b_const_g": lambda: (I.random_state(19, 11, 1, 31, mu=2e-3, kappa=3e-3, g=(0.3, -1.0, 0),
                                                     bc_type=((PER, PER), (FIX, REF), (0, 0)), bc_value=((0, 0), (1.5, 0), (0, 0))), 1, None),
    "2d_phi_periodic": lambda: (I.random_state(20, 10, 1, 32), 0, "periodic"),
    "2d_phi_walls_appendix_b": lambda: (I.random_state(17, 12, 1, 33, mu=1e-3, kappa=2e-3,
                                                       bc_type=((PER, PER), (REF, FIX), (0, 0)), bc_value=((0, 0), (0, 1.4), (0, 0))), 1, "walls"),
    "3d_appendix_b_const_g": lambda: (I.random_state(12, 9, 10, 34, mu=2e-3, kappa=3e-3, g=(0, 0, -1.0),
                                                     bc_type=((PER, PER), (PER, PER), (FIX, REF)), bc_value=((0, 0), (0, 0), (1.5, 0))), 1, None),
    "3d_phi_periodic_inviscid": lambda: (I.random_state(12, 9, 7, 35), 0, "periodic"),
    "3d_phi_walls_viscous": lambda: (I.random_state(10, 9, 9, 36, mu=1e-3, kappa=2e-3,
                                                    bc_type=((PER, PER), (REF, REF), (FIX, REF)), bc_value=((0, 0), (0, 0), (1.5, 0))), 0, "walls"),
    "3d_phi_walls_appendix_b": lambda: (I.random_state(9, 10, 8, 37, mu=1e-3, kappa=0.0,
                                                       bc_type=((REF, REF), (PER, PER), (REF, REF))), 1, "walls"),
}


@pytest.mark.parametrize("name", sorted(GEN_CASES))
def test_emulated_general_path_matches_oracle(name):
    (prm, U), eform, kind = GEN_CASES[name]()
    prm = dict(prm, energy_form=eform)
    if kind is not None:
        prm["phi"] = _phi_field(prm["nx"], prm["ny"], prm["nz"], prm["dx"], kind)
    _compare(prm, U, 3)
    if prm["nz"] > 1:
        _compare(prm, U, 2, zchunk=4)


def test_emulated_linear_potential_equals_constant_gravity():
    """An array Phi = -g.x must give the constant-g result up to the rounding of the potential differences."""
    prm, U = CASES["3d_all_walls_oblique_gravity"]()
    nx, ny, nz, h = prm["nx"], prm["ny"], prm["nz"], prm["dx"]
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    g = prm["g"]
    phi = -(g[0] * (i + 0.5) + g[1] * (j + 0.5) + g[2] * (k + 0.5)) * h
    dts = O.run(prm, U, 3, cfl=0.4)[1]
    A, _, _ = emu.run(prm, U, dts)
    B, _, _ = emu.run(dict(prm, phi=phi), U, dts)
    for f in range(5):
        assert np.abs(A[f] - B[f]).max() <= 1e-13 * np.abs(A[f]).max(), f
