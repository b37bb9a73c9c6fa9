"""C-ABI boundary (include/ark.h): the library builds for sm_100a, loads, exports every declared symbol and
validates its arguments.  No compute calls (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1903_09043_b200 import build
    build.build()
    from paper_1903_09043_b200 import binding
    return binding.load()


def test_exports_every_symbol_declared_in_header(lib):
    from paper_1903_09043_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "ark.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(ark_[a-z0-9_]+)\s*\(", hdr)))
    assert declared, "no declarations found"
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared


def test_version_and_workspace(lib):
    from paper_1903_09043_b200 import binding
    v = binding.version_string()
    assert "sm_100a" in v and "K=1.10" in v
    assert binding.workspace_bytes(3, 8, 1) == 0            # nx < 4
    assert binding.workspace_bytes(8, 8, 2) == 0            # nz must be 1 or >= 4
    b2 = binding.workspace_bytes(128, 128, 1)
    b3 = binding.workspace_bytes(64, 64, 64)
    assert b2 >= 2 * 4 * 132 * 132 * 8 and b3 >= 2 * 5 * 68 ** 3 * 8
    # 512^3: two padded states of 5 fields, ~11.3 GB, far below 180 GB
    assert 10e9 < binding.workspace_bytes(512, 512, 512) < 14e9


def test_size_queries_are_cheap_and_keep_the_documented_limits(lib):
    """ark_workspace_bytes / ark_potential_bytes / ark_halo_bytes are called per step by a slab run (binding caches them
    too): they must not run the z-chunk scheduling simulation of ark_create (milliseconds for 512^3)."""
    import time
    from paper_1903_09043_b200 import binding
    assert binding.workspace_bytes(4096, 4096, 1) == 0                 # more fused-step blocks than rate slots (ark.h)
    assert binding.workspace_bytes(2048, 2048, 1) > 0
    assert binding.workspace_bytes(1024, 1024, 1024) > 0
    assert lib.ark_halo_bytes(512, 512, 1) == 0 and lib.ark_potential_bytes(8, 8, 2) == 0
    assert lib.ark_halo_bytes(512, 512, 64) == 5 * 2 * 528 * 516 * 8   # 5 fields x 2 padded planes (pitch 528)
    t0 = time.perf_counter()
    for _ in range(200):
        lib.ark_halo_bytes(512, 512, 512)
        lib.ark_workspace_bytes(512, 512, 128)
    assert time.perf_counter() - t0 < 0.1                              # was 2 x 200 x ~10 ms


def test_create_rejects_bad_arguments_without_touching_the_gpu(lib):
    from paper_1903_09043_b200 import binding
    h = C.c_void_p()
    g = (C.c_double * 3)(0, 0, -1)
    bc = binding.ark_bc()
    ws = C.c_void_p(256)

    def create(nx=8, ny=8, nz=8, dx=0.1, gamma=1.4, mu=0.0, kappa=0.0, theta=1, bcp=bc, wsp=ws, nbytes=1 << 40):
        return lib.ark_create(C.byref(h), nx, ny, nz, dx, gamma, g, mu, kappa, theta,
                              C.byref(bcp) if bcp is not None else None, wsp, C.c_size_t(nbytes), None)

    assert create(nx=2) == binding.ARK_EINVAL
    assert create(nz=3) == binding.ARK_EINVAL
    assert create(dx=0.0) == binding.ARK_EINVAL
    assert create(gamma=1.0) == binding.ARK_EINVAL
    assert create(mu=-1.0) == binding.ARK_EINVAL
    assert create(theta=2) == binding.ARK_EINVAL
    assert create(wsp=None) == binding.ARK_EINVAL
    assert create(wsp=C.c_void_p(264)) == binding.ARK_EINVAL        # misaligned
    assert create(nbytes=1024) == binding.ARK_EINVAL                # too small
    bad = binding.ark_bc()
    bad.type[0][0] = binding.BC_PERIODIC
    bad.type[0][1] = binding.BC_REFLECTING
    assert create(bcp=bad) == binding.ARK_EINVAL                    # periodic on one side only
    bad2 = binding.ark_bc()
    bad2.type[2][0] = binding.BC_FIXED_T_WALL
    bad2.type[2][1] = binding.BC_REFLECTING
    bad2.value[2][0] = 0.0
    assert create(bcp=bad2) == binding.ARK_EINVAL                   # wall temperature must be positive
    assert b"ark_create" in lib.ark_last_error()
    assert h.value is None
    assert lib.ark_step(None, 0.1) == binding.ARK_EINVAL
    assert lib.ark_launch_count(None) == 0
    lib.ark_destroy(None)


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1903_09043_b200 import binding, inputs
    prm, U = inputs.random_state(8, 8, 1, 1)
    with pytest.raises(RuntimeError):
        binding.Solver(prm)
