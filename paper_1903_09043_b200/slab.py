"""Slab decomposition of a 3D domain along z over several GPUs.

PAPER.md:295 (section 3.2): "regular domain decomposition" with the "ghost-cell pattern ... per direction and side":
every sub-domain keeps ghost zones that hold the neighbouring sub-domain's cells.  Here the decomposition is 1-D along
the slowest axis (z): rank r owns planes [k0_r, k1_r) of the global grid, is an ordinary `binding.Solver` whose z sides
that face a neighbour are ARK_BC_EXTERNAL, and before every step
  1. hands out the two interior planes next to each such side (ark_get_halo; padded planes incl. x / y ghost cells),
  2. exchanges them with its neighbours (torch.distributed P2P: NCCL over NVLink / NVSwitch on a B200 node),
  3. stores the received planes into its ghost planes (ark_set_halo),
and the time step is the minimum over the ranks of ark_compute_dt (one all-reduce of one double).
Every per-cell operation is the single-domain one: the assembled state is bit-identical to the undivided run with the
strict build of the library (-DARK_STRICT --fmad=false) and within a few ulp (1e-14 relative) with the product build,
whose steady-state and boundary-plane code paths contract FMAs differently (tests/test_parity_gpu.py).

Status: `SlabSolver` over NCCL (the batch_isend_irecv exchange, its ordering against the solver stream, the all-reduce
of dt) has NOT run on hardware yet -- no multi-GPU box was available; what is verified is the index / exchange logic
(gloo, CPU) and the per-rank kernels (`LocalSlabs`, one GPU).

This module holds the host logic only (index arithmetic, neighbour ranks, the exchange); all arithmetic stays in the
kernels.  `partition`, `neighbours`, `local_params` and `exchange` have no CUDA dependency and are covered by the
world_size-2 gloo test on CPU; `SlabSolver` is the per-rank driver; `LocalSlabs` runs all sub-domains of a decomposition
inside ONE process on ONE GPU, one after the other (nothing waits on another launch), which is how the path is verified
on a single device.
"""
from . import inputs as I

BC_EXTERNAL = 4            # include/ark.h ARK_BC_EXTERNAL
MIN_PLANES = 4             # ark_create: nz >= 4


def partition(nz, world):
    """Plane range [k0, k1) of every rank: balanced contiguous slabs, the first nz % world ranks one plane thicker."""
    if world < 1 or nz < MIN_PLANES * world:
        raise ValueError("nz = %d cannot be split into %d slabs of at least %d planes" % (nz, world, MIN_PLANES))
    base, extra = divmod(nz, world)
    out, k = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((k, k + n))
        k += n
    return out


def neighbours(rank, world, periodic_z):
    """(rank below, rank above) or None where the slab ends at a physical z boundary."""
    if world == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (world - 1 if periodic_z else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic_z else None)
    return lo, hi


def local_params(prm, rank, world):
    """Parameters of rank `rank`'s sub-domain: its plane count and z boundary kinds (external towards neighbours, the
    global boundary condition at the physical ends).  Also returns its plane range (k0, k1)."""
    if int(prm["nz"]) <= 1:
        raise ValueError("slab decomposition needs a 3D grid")
    if prm.get("phi") is not None:
        raise ValueError("array-valued potentials are not available on sub-domains")
    k0, k1 = partition(int(prm["nz"]), world)[rank]
    periodic = int(prm["bc_type"][2][0]) == I.BC_PERIODIC
    lo, hi = neighbours(rank, world, periodic)
    bt = [list(map(int, row)) for row in prm["bc_type"]]
    bv = [list(map(float, row)) for row in prm["bc_value"]]
    if world > 1:
        if lo is not None:
            bt[2][0], bv[2][0] = BC_EXTERNAL, 0.0
        if hi is not None:
            bt[2][1], bv[2][1] = BC_EXTERNAL, 0.0
    p = dict(prm, nz=k1 - k0, bc_type=tuple(tuple(r) for r in bt), bc_value=tuple(tuple(r) for r in bv))
    return p, (k0, k1)


def exchange(dist, rank, world, periodic_z, send_lo, send_hi, recv_lo, recv_hi):
    """One halo exchange: my low planes go to the rank below (they become ITS high ghost planes), my high planes to the
    rank above; recv_lo / recv_hi receive my low / high ghost planes.  Tensors of equal size on the backend's device
    (CUDA for NCCL, CPU for gloo).  Non-blocking P2P batch, completed before returning.  With world == 2 and periodic z
    both neighbours are the same rank: the two messages are told apart by their order (ops of one pair are matched in
    the order they are posted: low-going first on both sides)."""
    lo, hi = neighbours(rank, world, periodic_z)
    ops = []
    # post in a global order that matches on both ends: every rank first talks "downwards" (send low / receive high),
    # then "upwards" (send high / receive low)
    if lo is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, lo))
    if hi is not None:
        ops.append(dist.P2POp(dist.irecv, recv_hi, hi))
    if hi is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, hi))
    if lo is not None:
        ops.append(dist.P2POp(dist.irecv, recv_lo, lo))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return lo, hi


class NonFiniteRate(RuntimeError):
    """the CFL rate of at least one sub-domain was not finite and positive (raised on EVERY rank)."""


def global_dt(dist, torch, local_dt, device="cpu"):
    """Minimum of the ranks' local time steps; local_dt is None on a rank whose own rate was invalid.  Such a rank must
    not leave before the collective (its peers would wait in the all-reduce for ever): it contributes the sentinel -1,
    which wins the MIN against every valid (positive) step, and then every rank raises NonFiniteRate together.
    (A NaN would not do: what MIN makes of a NaN differs between backends.)"""
    bad = local_dt is None or not (local_dt > 0.0) or local_dt == float("inf")
    t = torch.tensor([-1.0 if bad else float(local_dt)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    dt = float(t.item())
    if dt < 0.0:
        raise NonFiniteRate("ark_compute_dt: the maximum CFL rate of %s sub-domain is not finite and positive"
                            % ("this" if bad else "another"))
    return dt


class SlabSolver:
    """Rank-local driver of one slab: a binding.Solver plus the halo exchange and the global time step.

    prm: GLOBAL parameters; U_local: this rank's planes [k0, k1) of the dense state (5 CUDA tensors).  `dist` is
    torch.distributed with an initialised process group (NCCL), or None for world == 1."""

    def __init__(self, binding, prm, rank, world, dist=None, device="cuda:0"):
        import torch
        self.torch, self.dist, self.rank, self.world, self.binding = torch, dist, rank, world, binding
        self.prm_global = dict(prm)
        self.prm, (self.k0, self.k1) = local_params(prm, rank, world)
        self.periodic = int(prm["bc_type"][2][0]) == I.BC_PERIODIC
        self.s = binding.Solver(self.prm, device=device)
        self.lo, self.hi = neighbours(rank, world, self.periodic)
        n = self.s.halo_doubles()
        mk = lambda: torch.empty(n, dtype=torch.float64, device=self.s.device)
        self.send = [mk(), mk()]
        self.recv = [mk(), mk()]

    def set_state(self, U_local):
        self.s.set_state(U_local)

    def get_state(self):
        return self.s.get_state()

    def compute_dt(self, cfl):
        """min over the ranks of the local CFL step (= cfl / global max rate, the same double as on the undivided
        domain: a max over cells does not depend on the split).  A rank whose own rate is invalid still takes part in the
        all-reduce (see global_dt); all ranks then raise NonFiniteRate."""
        try:
            dt = self.s.compute_dt(cfl)
        except self.binding.ArkError as e:
            if e.code != self.binding.ARK_ENONFINITE:
                raise
            dt = None
        if self.dist is not None and self.world > 1:
            return global_dt(self.dist, self.torch, dt, self.s.device)
        if dt is None:
            raise NonFiniteRate("ark_compute_dt: the maximum CFL rate is not finite and positive")
        return dt

    def halo_exchange(self):
        if self.world == 1:
            return
        if self.lo is not None:
            self.s.get_halo(0, self.send[0])
        if self.hi is not None:
            self.s.get_halo(1, self.send[1])
        if self.dist.get_backend() != "nccl":
            # a backend that reads the buffers from the host side must see them finished; NCCL's P2P ops are enqueued
            # behind the current stream (the solver's) and `wait()` makes that stream wait for them: no host stall
            self.torch.cuda.current_stream(self.s.device).synchronize()
        exchange(self.dist, self.rank, self.world, self.periodic, self.send[0], self.send[1], self.recv[0], self.recv[1])
        if self.lo is not None:
            self.s.set_halo(0, self.recv[0])
        if self.hi is not None:
            self.s.set_halo(1, self.recv[1])

    def step(self, dt):
        self.halo_exchange()
        self.s.step(dt)

    def step_cfl(self, cfl):
        """One step of size cfl / (max over ALL ranks of the maximum CFL rate) with every number left on the device: the
        local rate (ark_max_rate_device), a MAX all-reduce of one double, the division, the halo exchange and the step
        (ark_step_device_dt) are all enqueued; the host never waits and never reads dt.  cfl / max rate is the same
        double ark_compute_dt forms on the host (IEEE division).  Nothing checks the rate: call compute_dt now and then."""
        t = self.torch
        if not hasattr(self, "_rate"):
            self._rate = t.empty(1, dtype=t.float64, device=self.s.device)
            self._dt = t.empty(1, dtype=t.float64, device=self.s.device)
            self._cfl = t.empty(1, dtype=t.float64, device=self.s.device)
        self._cfl.fill_(float(cfl))
        self.s.max_rate_device(self._rate)
        if self.dist is not None and self.world > 1:
            self.dist.all_reduce(self._rate, op=self.dist.ReduceOp.MAX)
        t.div(self._cfl, self._rate, out=self._dt)
        self.halo_exchange()
        self.s.step_device_dt(self._dt)

    def bytes_per_exchange(self):
        """bytes this rank sends per step (what must cross NVLink)."""
        return 8 * self.s.halo_doubles() * ((self.lo is not None) + (self.hi is not None))

    def close(self):
        self.s.close()


class LocalSlabs:
    """All sub-domains of a `world`-way decomposition inside one process on one GPU, stepped one after the other (no
    launch ever waits for another one): the single-device check of the slab path against the undivided solver."""

    def __init__(self, binding, prm, world, device="cuda:0"):
        self.world = world
        self.periodic = int(prm["bc_type"][2][0]) == I.BC_PERIODIC
        self.parts = [local_params(prm, r, world) for r in range(world)]
        self.solvers = [binding.Solver(p, device=device) for p, _ in self.parts]
        self.nxy = int(prm["nx"]) * int(prm["ny"])

    def set_state(self, U):
        """U: the GLOBAL dense state (5 flat CUDA tensors, x fastest)."""
        for s, (_, (k0, k1)) in zip(self.solvers, self.parts):
            s.set_state([a[k0 * self.nxy:k1 * self.nxy].contiguous() for a in U])

    def get_state(self):
        import torch
        parts = [s.get_state() for s in self.solvers]
        return [torch.cat([p[f] for p in parts]) for f in range(5)]

    def compute_dt(self, cfl):
        return min(s.compute_dt(cfl) for s in self.solvers)

    def _exchange(self):
        if self.world > 1:
            halos = [(s.get_halo(0), s.get_halo(1)) for s in self.solvers]
            for r, s in enumerate(self.solvers):
                lo, hi = neighbours(r, self.world, self.periodic)
                if lo is not None:
                    s.set_halo(0, halos[lo][1])      # my low ghost planes = the high planes of the rank below
                if hi is not None:
                    s.set_halo(1, halos[hi][0])

    def step(self, dt):
        self._exchange()
        for s in self.solvers:
            s.step(dt)

    def step_cfl(self, cfl):
        """The device-side loop of SlabSolver.step_cfl on one GPU: per-slab rates -> max -> dt = cfl / max, all in device
        memory; no call of this method waits for the GPU or reads a number back."""
        import torch
        dev = self.solvers[0].device
        if not hasattr(self, "_rates"):
            self._rates = torch.empty(self.world, dtype=torch.float64, device=dev)
            self._rate = torch.empty(1, dtype=torch.float64, device=dev)
            self._dt = torch.empty(1, dtype=torch.float64, device=dev)
            self._cfl = torch.empty(1, dtype=torch.float64, device=dev)
        self._cfl.fill_(float(cfl))
        for r, s in enumerate(self.solvers):
            s.max_rate_device(self._rates[r:r + 1])
        torch.amax(self._rates, dim=0, keepdim=True, out=self._rate)
        torch.div(self._cfl, self._rate, out=self._dt)
        self._exchange()
        for s in self.solvers:
            s.step_device_dt(self._dt)

    def close(self):
        for s in self.solvers:
            s.close()
