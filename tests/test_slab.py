"""Slab decomposition along z (PAPER.md:295 regular domain decomposition with ghost zones,
:303-307): host logic on CPU.  world_size-2 / -3 gloo processes exchange halo planes with the functions the GPU driver
uses (paper_1903_09043_b200/slab.py: partition, neighbours, local_params, exchange) and every rank's padded slab must be
bit-identical to the corresponding planes of the ORACLE's ghost-filled undivided domain.  The GPU side of the path
(ARK_BC_EXTERNAL, ark_get_halo / ark_set_halo) is tested in test_parity_gpu.py on one device."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1903_09043_b200 import inputs as I  # noqa: E402
from paper_1903_09043_b200 import slab  # noqa: E402

PER, REF, FIX = I.BC_PERIODIC, I.BC_REFLECTING, I.BC_FIXED_T


def test_partition_is_contiguous_balanced_and_complete():
    for nz, world in ((512, 8), (13, 3), (16, 4), (257, 8), (4, 1)):
        parts = slab.partition(nz, world)
        assert parts[0][0] == 0 and parts[-1][1] == nz and len(parts) == world
        for (a0, a1), (b0, b1) in zip(parts, parts[1:]):
            assert a1 == b0
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1 and min(sizes) >= slab.MIN_PLANES
    with pytest.raises(ValueError):
        slab.partition(15, 4)                       # a slab would be thinner than the solver's minimum of 4 planes


def test_neighbours_and_local_boundary_kinds():
    assert slab.neighbours(0, 1, True) == (None, None)
    assert slab.neighbours(0, 4, False) == (None, 1) and slab.neighbours(3, 4, False) == (2, None)
    assert slab.neighbours(0, 4, True) == (3, 1) and slab.neighbours(3, 4, True) == (2, 0)
    assert slab.neighbours(0, 2, True) == (1, 1)
    prm, _ = I.random_state(8, 8, 16, 1, bc_type=((PER, PER), (PER, PER), (FIX, REF)), bc_value=((0, 0), (0, 0), (1.5, 0)))
    p0, r0 = slab.local_params(prm, 0, 3)
    p1, r1 = slab.local_params(prm, 1, 3)
    p2, r2 = slab.local_params(prm, 2, 3)
    assert (r0, r1, r2) == ((0, 6), (6, 11), (11, 16)) and (p0["nz"], p1["nz"], p2["nz"]) == (6, 5, 5)
    assert p0["bc_type"][2] == (FIX, slab.BC_EXTERNAL) and p0["bc_value"][2][0] == 1.5
    assert p1["bc_type"][2] == (slab.BC_EXTERNAL, slab.BC_EXTERNAL)
    assert p2["bc_type"][2] == (slab.BC_EXTERNAL, REF)
    assert p1["bc_type"][0] == (PER, PER) and p1["nx"] == 8
    pp, _ = slab.local_params(dict(prm, bc_type=((PER, PER), (PER, PER), (PER, PER))), 0, 2)
    assert pp["bc_type"][2] == (slab.BC_EXTERNAL, slab.BC_EXTERNAL)
    same, rr = slab.local_params(prm, 0, 1)
    assert same["bc_type"][2] == (FIX, REF) and rr == (0, 16)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _case(periodic):
    zbc = (PER, PER) if periodic else (FIX, REF)
    return I.random_state(9, 8, 14, 77, mu=1e-3, kappa=2e-3, g=(0, 0, -1.0),
                          bc_type=((PER, PER), (REF, REF), zbc), bc_value=((0, 0), (0, 0), (1.5, 0) if not periodic else (0, 0)))


def _worker(rank, world, port, periodic, out):
    sys.path.insert(0, ROOT)
    from oracle import ark_oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        prm, U = _case(periodic)
        G = O.fill_ghosts(prm, U)                                        # the undivided domain, ghost-filled
        lp, (k0, k1) = slab.local_params(prm, rank, world)
        Ul = [np.asarray(a)[k0:k1] for a in U]
        # the oracle knows no external side: a reflecting stand-in there; only the planes that do NOT depend on it are used
        bt = [list(r) for r in lp["bc_type"]]
        ext = [bt[2][s] == slab.BC_EXTERNAL for s in range(2)]
        for s in range(2):
            if ext[s]:
                bt[2][s] = REF
        if bt[2][0] == PER or bt[2][1] == PER:
            bt[2] = [REF, REF]
        L = O.fill_ghosts(dict(lp, bc_type=bt), Ul)                      # interior planes with x / y ghosts (+ physical z walls)
        L = np.stack(L)                                                  # (5, nzl+4, ny+4, nx+4)
        send_lo = torch.from_numpy(np.ascontiguousarray(L[:, 2:4]))
        send_hi = torch.from_numpy(np.ascontiguousarray(L[:, -4:-2]))
        recv_lo, recv_hi = torch.zeros_like(send_lo), torch.zeros_like(send_hi)
        lo, hi = slab.exchange(dist, rank, world, periodic, send_lo, send_hi, recv_lo, recv_hi)
        assert (lo is not None) == ext[0] and (hi is not None) == ext[1]
        if lo is not None:
            L[:, 0:2] = recv_lo.numpy()
        if hi is not None:
            L[:, -2:] = recv_hi.numpy()
        ref = np.stack(G)[:, k0:k1 + 4]
        # ghost planes beyond a physical wall only exist on the end ranks; there the local wall fill must agree as well
        ok = bool(np.array_equal(L, ref))
        worst = float(np.abs(L - ref).max())
        res = torch.tensor([1.0 if ok else 0.0, worst], dtype=torch.float64)
        gathered = [torch.zeros_like(res) for _ in range(world)]
        dist.all_gather(gathered, res)
        if rank == 0:
            out.put([g.tolist() for g in gathered])
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True), (3, False)])
def test_halo_exchange_reproduces_the_undivided_ghost_fill(world, periodic):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, periodic, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for ok, worst in res:
        assert ok == 1.0, (world, periodic, worst)


def _dt_worker(rank, world, port, bad_rank, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local = [0.25, 0.125, 0.5][rank]
        got = slab.global_dt(dist, torch, local)                            # every rank valid: the minimum, exactly
        try:
            slab.global_dt(dist, torch, None if rank == bad_rank else local)
            raised = ""
        except slab.NonFiniteRate as e:
            raised = str(e)
        after = slab.global_dt(dist, torch, local)                          # nobody is left behind in a collective
        out.put((rank, got, raised, after))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,bad_rank", [(2, 1), (3, 0)])
def test_invalid_rate_on_one_rank_raises_on_all_ranks_and_nobody_hangs(world, bad_rank):
    """a rank whose ark_compute_dt fails must still enter the dt all-reduce, otherwise its peers hang."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_dt_worker, args=(r, world, port, bad_rank, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = min([0.25, 0.125, 0.5][:world])
    for rank, got, raised, after in res:
        assert got == want and after == want
        assert ("this" if rank == bad_rank else "another") in raised, (rank, raised)
