"""Seeded input generators (paper_1903_09043_b200/inputs.py): determinism, numpy/torch agreement, per-cell
regeneration of sub-boxes, and the discrete hydrostatic relation (14) of the initial columns."""
import numpy as np
import pytest
import torch

from paper_1903_09043_b200 import inputs as I


def test_uniform01_is_counter_based_and_matches_torch():
    c = np.arange(0, 4096, dtype=np.int64)
    a = I.uniform01(1234, c)
    b = I.uniform01(1234, torch.arange(0, 4096, dtype=torch.int64)).numpy()
    assert np.array_equal(a, b)
    assert a.min() >= 0.0 and a.max() < 1.0
    assert abs(a.mean() - 0.5) < 0.02 and abs(a.var() - 1.0 / 12.0) < 0.01
    assert np.array_equal(I.uniform01(1234, c[100:200]), a[100:200])        # stateless
    assert not np.array_equal(I.uniform01(1235, c), a)
    big = I.uniform01(7, np.array([2 ** 40 + 3, 2 ** 62], dtype=np.int64))
    assert np.all((big >= 0) & (big < 1))


def test_torch_and_numpy_builders_agree():
    for build in (lambda d: I.config1_atmosphere(16, device=d), lambda d: I.config3_rb2d(16, 12, device=d),
                  lambda d: I.config4_rb3d(8, device=d), lambda d: I.config5_convection3d(8, device=d),
                  lambda d: I.config2_gresho(16, device=d)):
        pn, Un = build(None)
        pt, Ut = build("cpu")
        assert pn == pt
        for a, b in zip(Un, Ut):
            assert (a is None) == (b is None)
            if a is not None:
                assert np.array_equal(np.asarray(a).reshape(-1), b.numpy().reshape(-1))


def test_sub_box_regeneration():
    prm, U = I.config5_convection3d(12)
    box = ((3, 9), (2, 7), (4, 12))
    prm_b, Ub = I.config5_convection3d(12, box=box)
    assert prm == prm_b
    for a, b in zip(U, Ub):
        assert np.array_equal(a[3:9, 2:7, 4:12], b)


def test_columns_satisfy_discrete_hydrostatic_relation():
    h = 1.0 / 64
    T, rho = I.polytrope(64, h, 0.57, 0.9, 0.1)
    p = rho * T
    lhs = p[1:] - p[:-1]
    rhs = -0.5 * (rho[1:] + rho[:-1]) * h
    assert np.abs(lhs - rhs).max() < 1e-15
    prm, U = I.config5_convection3d(16)
    assert U[0].max() / U[0].min() > 15          # steep stratification (chi = 100 wall to wall; cell centres see less)
    # heated from below at 10 x the conductive flux kappa*beta (beta = 1/(m+1) = 0.5), insulating top
    assert prm["bc_type"][2] == (I.BC_FLUX, I.BC_REFLECTING) and prm["mu"] == 1e-4
    assert abs(prm["bc_value"][2][0] - 10 * 2.5e-4 * 0.5) < 1e-15
    assert I.config5_convection3d(16, heat=0.0)[0]["bc_type"][2] == (I.BC_REFLECTING, I.BC_REFLECTING)
    prm, U = I.config4_rb3d(8)
    assert abs(prm["mu"] - 7.473e-4) < 2e-6 and abs(prm["kappa"] - 1.8683e-3) < 5e-6
    prm, U = I.config3_rb2d(16, 8)
    assert abs(prm["mu"] - 1.8544e-3) < 2e-6 and abs(prm["kappa"] - 4.6361e-3) < 5e-6


def test_second_workloads_follow_the_paper():
    """Rayleigh-Taylor and the chi = 21 layer."""
    prm, U = I.rayleigh_taylor(20, 60)
    assert (prm["nx"], prm["ny"], prm["nz"]) == (20, 60, 1) and abs(prm["dx"] - 0.5 / 20) < 1e-16
    rho = U[0][0]
    assert (rho[:30] == 1.0).all() and (rho[30:] == 2.0).all()                 # rho = 1 for y < 0, 2 for y >= 0
    v = U[2][0] / rho
    assert abs(v.max() - 0.01 * np.cos(np.pi * 0.5 / 20) ** 2 * np.cos(np.pi * 0.5 / 60) ** 2) < 1e-12   # C/4 (1+cos)(1+cos) near the centre
    assert v.min() >= 0.0 and np.abs(U[1]).max() == 0.0
    p = 0.4 * (U[4][0] - 0.5 * rho * v * v)
    h = prm["dx"]
    lhs = p[1:, 0] - p[:-1, 0]                                                  # discrete balance (14) holds on every face
    rhs = -0.5 * (rho[1:, 0] + rho[:-1, 0]) * 0.1 * h
    assert np.abs(lhs - rhs).max() < 1e-15
    with pytest.raises(ValueError):
        I.rayleigh_taylor(20, 50)
    prm, U = I.rb2d_chi21(16, 64)
    assert prm["bc_type"][1] == (I.BC_FLUX, I.BC_FIXED_T)
    beta = 1.0 / 2.3
    assert abs(prm["bc_value"][1][0] - prm["kappa"] * beta) < 1e-16           # the polytrope's own conductive flux
    T_top = prm["bc_value"][1][1]
    assert abs(((T_top + beta) / T_top) ** 1.3 - 21.0) < 1e-10                 # chi = 21 wall to wall
