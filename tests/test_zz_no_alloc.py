"""ark_cfl_dt_static: the CFL time step for callers that cannot allocate device memory (include/ark.h).

Who needs it: a caller that holds the five dense fields on the GPU but has no way to obtain a solver workspace -- a
coupling / in-situ plug-in inside an application whose own pool already owns the device's memory, or a time loop that
must not trigger the device-wide synchronisation of cudaMalloc / cudaFree.  The entry point keeps the reduction's
per-block scratch in a fixed 256 KiB array inside the library (limit: 2^27 cells) and allocates nothing.

What is checked: its output against the existing path (Solver.set_state + ark_compute_dt, whose scratch lives in the
caller-allocated workspace) within the 1e-13 the compute_dt tests use, on calls IN A ROW that share the library's one
scratch array -- first a grid with many blocks and a high rate, then a smaller grid with a lower rate, whose result
would be wrong if slots left over from the first call were read -- and that grids beyond the limit are refused.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide other tests); the
GPU test passes both alone in a fresh process (its first call then does the once-per-device address look-up) and
after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_1903_09043_b200 import inputs as I


@pytest.fixture(scope="module")
def B():
    from paper_1903_09043_b200 import build
    build.build()
    from paper_1903_09043_b200 import binding
    binding.load()
    return binding


def _dev(U):
    return [None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).reshape(-1).cuda() for a in U]


def _existing_path(B, prm, Ud, cfl):
    """max rate and dt through the solver handle: padded copy + two-pass reduction in the caller's workspace."""
    s = B.Solver(prm)
    s.set_state(Ud)
    dt = s.compute_dt(cfl)
    s.close()
    return dt


def test_limit_is_stated_and_enforced_before_any_gpu_work(B):
    """No GPU needed: argument checks come before the first CUDA call."""
    lib = B.load()
    assert B.cfl_dt_static_max_cells() == 2 ** 27 == 512 ** 3
    p = C.c_void_p(256)                                       # never dereferenced: the call is refused first

    def call(nx, ny, nz, dx=0.1, gamma=1.4, mu=0.0, kappa=0.0, cfl=0.4, rho=p, rhow=p, out=p):
        return lib.ark_cfl_dt_static(nx, ny, nz, dx, gamma, mu, kappa, rho, p, p, rhow, p, cfl, out, None)

    assert call(1024, 512, 512) == B.ARK_EINVAL               # 2^28 cells: twice the limit
    msg = lib.ark_last_error().decode()
    assert "134217728" in msg and "ark_compute_dt" in msg, msg
    assert call(513, 512, 512) == B.ARK_EINVAL                # just above 512^3
    assert call(3, 8, 8) == B.ARK_EINVAL and call(8, 8, 2) == B.ARK_EINVAL
    assert call(8, 8, 8, dx=0.0) == B.ARK_EINVAL and call(8, 8, 8, gamma=1.0) == B.ARK_EINVAL
    assert call(8, 8, 8, cfl=0.0) == B.ARK_EINVAL and call(8, 8, 8, mu=-1.0) == B.ARK_EINVAL
    assert call(8, 8, 8, rho=None) == B.ARK_EINVAL and call(8, 8, 8, out=None) == B.ARK_EINVAL
    assert call(8, 8, 8, rhow=None) == B.ARK_EINVAL           # 3D needs rho*w ...
    # ... 2D does not (NULL rhow passes validation); not called here because it would go on to launch


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_calls_in_a_row(B):
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cfl = 0.4
    # call order matters: many blocks / fast state first, then fewer blocks with lower rates, then the first again
    cases = [
        ("3d_walls_viscous_72x40x56", I.random_state(72, 40, 56, 31, g=(0.0, 0.0, -1.5), mu=2e-3, kappa=3e-3,
                                                     bc_type=((0, 0), (0, 0), (I.BC_REFLECTING, I.BC_REFLECTING)))),
        ("config1_atmosphere_64", I.config1_atmosphere(64)),                       # 2D, 1 block, nearly at rest
        ("config4_rb3d_40", I.config4_rb3d(40)),
        ("2d_ragged_130x67", I.random_state(130, 67, 1, 32)),
    ]
    cases.append(cases[0])
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    got = []
    dev_states = [(name, prm, _dev(U)) for name, (prm, U) in cases]
    for name, prm, Ud in dev_states:                          # the static-scratch calls, back to back on one stream
        B.cfl_dt_static(prm, Ud, cfl, out)
        got.append(out.cpu().numpy().copy())
    rates = [g[0] for g in got]
    assert rates[1] < 0.5 * rates[0], "the second case must have the lower rate for the stale-slot check to bite"
    for (name, prm, Ud), g in zip(dev_states, got):
        dt_ref = _existing_path(B, prm, Ud, cfl)
        assert np.isfinite(g).all() and g[0] > 0.0, (name, g)
        assert abs(g[1] - dt_ref) <= 1e-13 * dt_ref, (name, g[1], dt_ref)
        assert abs(g[0] - cfl / dt_ref) <= 1e-13 * g[0], (name, g[0], cfl / dt_ref)
    assert np.array_equal(got[0], got[-1])                    # same input, same bits, whatever ran in between
    # a state without a valid rate comes back as a NaN in d_out (nothing is synchronised or checked on the host)
    name, prm, Ud = dev_states[2]
    bad = [a.clone() for a in Ud]
    bad[4][1234] = -5.0                                       # negative pressure -> NaN sound speed
    B.cfl_dt_static(prm, bad, cfl, out)
    assert not np.isfinite(out.cpu().numpy()[0])
    B.cfl_dt_static(prm, Ud, cfl, out)                        # and the next call is clean again
    assert np.array_equal(out.cpu().numpy(), got[2])
