/* ark.h -- C ABI of the B200-native (sm_100a) hot path of the ARK all-Mach solver (arXiv 1903.09043).
 *
 * One explicit finite-volume time step of the stratified compressible Euler / Navier-Stokes equations on a
 * uniform 2D/3D Cartesian grid, fp64, single GPU:
 *   ghost-cell fill -> acoustic step (u*, Pi*, L~, U~) -> transport step (upwind on u*) + viscous / heat
 *   face fluxes -> conservative update, plus the CFL time-step max-reduction.
 * "PAPER.md:<n>" cites /root/reference/PAPER.md; "A<n>" are the readings listed in DESIGN.md.
 *
 * Conventions
 *   - All state arrays are DENSE interior-only fp64, nx*ny*nz elements, x fastest:
 *       idx = i + nx*(j + ny*k).  rho, rho*u, rho*v, rho*w, E  with  E = rho*e + 1/2 rho |u|^2
 *       (total energy density WITHOUT potential energy).
 *   - nz == 1 selects 2D: the z axis and rho*w do not exist; rhow may be NULL.
 *   - Pointers are DEVICE pointers unless the function name ends in _host.  The caller owns every
 *     array it passes; the library copies into / out of its own padded SoA buffers and never
 *     retains a caller pointer except the workspace.
 *   - The workspace is caller-allocated device memory (PyTorch in this repo) of at least
 *     ark_workspace_bytes() bytes, 256-byte aligned; it must outlive the handle.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).  Every call
 *     enqueues on that stream; only the calls documented as synchronising wait for it.
 *   - A handle belongs to the CUDA device that was current in ark_create (its workspace, stream and kernel
 *     attributes live there): calling an entry point while another device is current returns ARK_EINVAL.
 *   - Every entry point returns an ARK_* code and never throws; ark_last_error() gives a text for
 *     the last failure on the calling thread.
 *   - Gravity is the constant vector g (Phi = -g.x, never stored: A12) unless ark_set_potential supplies an array.
 *     The acoustic impedance
 *     constant is K = 1.1 (a = K max(rho_L c_L, rho_R c_R), A2), reported by
 *     ark_version_string().
 */
#ifndef ARK_H
#define ARK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ark_solver ark_solver; /* opaque, owned by the library */

enum { ARK_OK = 0, ARK_EINVAL = -1, ARK_ENOMEM = -2, ARK_ECUDA = -3, ARK_ENONFINITE = -4 };

/* Boundary kinds (A9; PAPER.md:295 ghost zones, :378 reflecting + hydrostatic extrapolation,
 * :457 fixed temperature, :435 imposed temperature flux).  Periodic must be set on both sides of an axis. */
enum { ARK_BC_PERIODIC = 0, ARK_BC_REFLECTING = 1, ARK_BC_FIXED_T_WALL = 2, ARK_BC_FLUX_WALL = 3,
       /* ghost zones that hold a neighbouring sub-domain's cells (regular domain decomposition): z axis of 3D
        * grids only; the library never fills them, the caller does with ark_set_halo before every ark_step */
       ARK_BC_EXTERNAL = 4 };

typedef struct {
    int type[3][2];     /* [axis x,y,z][lo,hi] */
    double value[3][2]; /* ARK_BC_FIXED_T_WALL: wall temperature (T = p/rho, A8).  ARK_BC_FLUX_WALL (PAPER.md:435,
                           A22): conductive heat flux ENTERING the domain through this wall, any sign; the velocity
                           is reflected as at a reflecting wall; needs kappa > 0.  Ignored otherwise. */
} ark_bc;

/* Bytes of device workspace ark_create needs for an nx*ny*nz grid; 0 if the sizes are invalid (nx,ny >= 4, nz == 1 or
 * >= 4, each <= 16384) or if the grid needs more fused-step blocks than the per-block rate scratch holds (58 432:
 * e.g. 2D 4096^2 is too large, 2D 2048^2 and 3D 1024^3 fit); ark_create rejects the same grids with ARK_EINVAL. */
size_t ark_workspace_bytes(int nx, int ny, int nz);

/* Create a solver.  nx,ny >= 4; nz >= 4 or nz == 1 (2D).  dx > 0 (uniform); gamma > 1
 * (ideal gas); g[3] constant gravity; mu, kappa >= 0 constant dynamic
 * viscosity and conductivity; low_mach_theta: 0 -> theta == 1, 1 -> eq. (13)
 * (PAPER.md:218-222, 325).  d_workspace: device memory of the CURRENT device, see above.  Errors: ARK_EINVAL (bad
 * argument, workspace too small, misaligned or not memory of the current device), ARK_ECUDA. */
int ark_create(ark_solver** out, int nx, int ny, int nz, double dx, double gamma, const double g[3],
               double mu, double kappa, int low_mach_theta, const ark_bc* bc,
               void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Copy a dense device state into the solver (asynchronous on the stream). */
int ark_set_state(ark_solver*, const double* rho, const double* rhou, const double* rhov,
                  const double* rhow, const double* E);
/* Copy the current state out to dense device arrays (asynchronous on the stream). */
int ark_get_state(ark_solver*, double* rho, double* rhou, double* rhov, double* rhow, double* E);

/* Same with HOST arrays (pageable or pinned).  The copies run on the stream through a staging
 * area inside the workspace; both calls return after the stream has been synchronised. */
int ark_set_state_host(ark_solver*, const double* rho, const double* rhou, const double* rhov,
                       const double* rhow, const double* E);
int ark_get_state_host(ark_solver*, double* rho, double* rhou, double* rhov, double* rhow, double* E);

/* CFL time step ("time step kernel"; formula = A4):
 *   dt = cfl / max_c [ sum_d (|u_d| + c)/dx + 2 ndim max(4 mu/3, (gamma-1) kappa) / (rho dx^2) ].
 * Deterministic two-pass max reduction (NaN-propagating).  Synchronises the stream (16-byte D2H).
 * Returns ARK_ENONFINITE if the maximum rate is not finite and positive. */
int ark_compute_dt(ark_solver*, double cfl, double* dt_out);

/* The same CFL time step for callers that cannot allocate device memory: no handle, no workspace, no cudaMalloc /
 * cudaFree / cudaMallocHost and no allocating library routine anywhere on this path.
 *
 * Who that is: every other entry point needs an ark_solver, and a solver needs a workspace of ark_workspace_bytes() that
 * somebody must allocate (two padded copies of the state).  A code that only wants to ask "what time step would ARK take
 * on this state?" -- a coupling or in-situ analysis plug-in running inside a host application whose own memory pool has
 * already claimed the GPU, or a time loop that must not pay the device-wide synchronisation cudaMalloc and cudaFree imply
 * -- has the five dense fields on the device and nowhere to put a workspace.  Here the only scratch the reduction needs
 * (one double per block of its first pass) lives inside the library image: a static 256 KiB device array that each GPU
 * which loads the library holds until the process exits.
 *
 * rho .. E: DEVICE, dense interior-only fields as everywhere in this header (nx*ny*nz doubles, x fastest; rhow may be NULL
 * when nz == 1), read in place, never copied.  d_out: DEVICE, 2 doubles, written as { max rate, cfl / max rate } with the
 * rate of ark_compute_dt (reading A4).  Asynchronous on cuda_stream; nothing is synchronised and nothing is checked on
 * the host, so a state without a finite positive maximum rate shows as a NaN / non-positive d_out[0] (NaN-propagating
 * max), not as ARK_ENONFINITE.
 *
 * Limit: nx*ny*nz <= ark_cfl_dt_static_max_cells() = 2^27 = 134 217 728 cells (512^3: 32 768 scratch slots x 4096 cells
 * per block).  Larger grids are rejected with ARK_EINVAL before anything is launched; use ark_compute_dt for them.
 *
 * First call on a device: the library looks up the device address of its scratch array for the device that is current
 * (once per device, cached).  Make that first call outside any stream capture; later calls only launch two kernels.
 *
 * Sharing: there is ONE scratch array per GPU, shared by every call from every thread and stream, and it keeps whatever
 * the previous call left in it.  Nothing in it has to start at zero -- each call overwrites the slots it is going to
 * read before reading them, so a smaller grid after a larger one is safe -- but two calls that are in flight on the same
 * GPU at the same time (different streams, or different host threads on streams that are not ordered with each other)
 * race on the array and may both return garbage.  Order them (same stream, or events).
 * Errors: ARK_EINVAL (sizes as for ark_create, too many cells, dx/gamma/mu/kappa/cfl out of range, NULL pointer),
 * ARK_ECUDA. */
size_t ark_cfl_dt_static_max_cells(void);
int ark_cfl_dt_static(int nx, int ny, int nz, double dx, double gamma, double mu, double kappa,
                      const double* rho, const double* rhou, const double* rhov, const double* rhow, const double* E,
                      double cfl, double* d_out, void* cuda_stream);

/* Advance the state by one full step of size dt (ghost fill, acoustic + transport + dissipative
 * fluxes, conservative update).  Asynchronous on the stream. */
int ark_step(ark_solver*, double dt);

/* The two halves of { ark_compute_dt ; ark_step } with the numbers kept in DEVICE memory, for time loops in which the step
 * size depends on more than this solver and the host must not wait for the GPU: a slab decomposition
 * takes dt = cfl / (max over the sub-domains' maximum rates), which a collective can form on device memory.
 * ark_max_rate_device writes the maximum CFL rate of the current state (the quantity ark_compute_dt divides cfl by) to
 * d_rate_out (1 double); ark_step_device_dt advances the state by the step size found in d_dt (1 double) when the
 * kernels run.  Both are asynchronous on the stream and check nothing on the host: a rate that is not finite and positive
 * simply propagates (NaN state); call ark_compute_dt from time to time to detect that.  Errors: ARK_EINVAL, ARK_ECUDA. */
int ark_max_rate_device(ark_solver*, double* d_rate_out);
int ark_step_device_dt(ark_solver*, const double* d_dt);

/* Convenience: nsteps x { dt = cfl / max rate ; step(dt) } with the time step kept on the device
 * (no host round trip per step).  If dts_out (HOST, nsteps doubles) is not NULL the step sizes are
 * copied there.  The call synchronises the stream ONCE, after the last step, to read a sticky device-side flag:
 * it returns ARK_ENONFINITE if any maximum rate of the run was not finite and positive (the remaining steps of such a
 * run have consumed a NaN step size; the state is then meaningless), with or without dts_out.
 * After the first step, pairs of steps are replayed from a CUDA graph captured on a stream of the library's own
 * (ordered with the caller's stream through events): the small 2D configurations are launch-latency-bound. */
int ark_run(ark_solver*, int nsteps, double cfl, double* dts_out);

/* Energy update (PAPER.md:194-210 and Appendix B, :514-546).  ARK_ENERGY_CONSERVATIVE (default): rho*E advanced in
 * flux form with the mass-flux-weighted gravity work, which conserves sum (E + rho Phi) to
 * round-off.  ARK_ENERGY_APPENDIX_B: the non-conservative scheme of Appendix B; mass and momentum are unchanged, the
 * energy carries the source (dt/dx) (uS)_i, (uS)_i = 1/2 (u*_{i+1/2} S_{i+1/2} + u*_{i-1/2} S_{i-1/2}) summed over the
 * axes, in the acoustic and in the final update (reading A24 of DESIGN.md).  Takes effect at the
 * next step.  Errors: ARK_EINVAL. */
enum { ARK_ENERGY_CONSERVATIVE = 0, ARK_ENERGY_APPENDIX_B = 1 };
int ark_set_energy_form(ark_solver*, int form);

/* Array-valued gravitational potential Phi(x) (S_{i+1/2} = -1/2 (rho_i + rho_{i+1}) (Phi_{i+1} - Phi_i),
 * PAPER.md:152; gravity work with the upwind potential; ghost-cell density from relation (14) with the
 * potential difference).  d_phi: DEVICE array, dense interior values at the cell centres (nx*ny*nz, x
 * fastest), copied; ghost values (reading A25): periodic axes wrap, wall axes continue Phi linearly, which reproduces a
 * constant gravity exactly.  d_buffer: caller-allocated DEVICE memory of at least ark_potential_bytes(nx, ny, nz) bytes,
 * 256-byte aligned, which the library keeps using (padded potential) until ark_destroy or the next ark_set_potential; the
 * caller owns it.  While a potential is set, the vector g of ark_create is ignored and ark_diagnostics uses Phi for the
 * total energy.  d_phi == NULL returns to the constant g (buffer ignored).  Algorithmic traffic of a step rises from 80
 * to 88 B per cell update in 3D (64 -> 72 B in 2D).  Asynchronous on the stream.  Errors: ARK_EINVAL, ARK_ECUDA. */
size_t ark_potential_bytes(int nx, int ny, int nz);
int ark_set_potential(ark_solver*, const double* d_phi, void* d_buffer, size_t buffer_bytes);

/* Slab decomposition along z (PAPER.md:295 "regular domain decomposition ... ghost-cell pattern", :303-307): a
 * sub-domain is an ordinary solver whose z sides that face a neighbour are ARK_BC_EXTERNAL.  Before every step each
 * sub-domain hands out the two interior planes next to such a side (ark_get_halo) and receives the neighbour's into its
 * ghost planes (ark_set_halo); the time step is the minimum of the sub-domains' ark_compute_dt.  A halo is
 * ark_halo_bytes() bytes of DEVICE memory: [field][2 planes][ny+4 rows][row pitch], i.e. padded planes WITH their x / y
 * ghost cells (ark_get_halo runs the x and y ghost sweeps first; the following ark_step does not repeat them), so that every
 * cell sees the same neighbourhood as on the undivided domain: the assembled result is bit-identical to it in the strict
 * build (-DARK_STRICT --fmad=false) and within a few ulp (1e-14 relative) in the product build, whose steady-state and
 * boundary-plane code paths contract FMAs differently.  side: 0 = low z, 1 = high z.  Both calls are asynchronous
 * on the stream; ark_get_halo is accepted on any 3D solver and side (a physical wall side simply hands out its interior
 * planes; slab.LocalSlabs relies on it), ark_set_halo only on ARK_BC_EXTERNAL sides; the caller moves the buffers between devices (NCCL send/recv or peer copies over NVLink).  ark_run and
 * array-valued potentials are not available on sub-domains.  Errors: ARK_EINVAL (2D solver, bad side, side not
 * external), ARK_ECUDA. */
size_t ark_halo_bytes(int nx, int ny, int nz);
int ark_get_halo(ark_solver*, int side, double* d_buf);
int ark_set_halo(ark_solver*, int side, const double* d_buf);

/* Diagnostics of the current state as the paper reports them (PAPER.md:398-407 maximum velocity, :435 mean absolute
 * velocity, :14 conserved mass and total energy).  out (HOST, 6 doubles) = { max |u|, mean |u|, kinetic energy
 * sum 1/2 rho |u|^2 dV, max Mach number |u|/c, mass sum rho dV, total energy sum (E + rho Phi) dV } with Phi = -g.x
 * at the cell centres and dV = dx^ndim.  Two-pass reduction without atomics (bit-reproducible); synchronises. */
int ark_diagnostics(ark_solver*, double* out);

/* Kinetic-energy power spectrum of the horizontal middle plane (Fig. 11; reading A26): plane k = nz/2,
 * w_c = sqrt(rho) u_c, w^_c(kx,ky) = 1/(nx ny) sum w_c exp(-2 pi i (kx i/nx + ky j/ny)); out[kappa] = sum over the shell
 * floor(|k~| + 1/2) == kappa (signed wavenumbers) of 1/2 sum_c |w^_c|^2, kappa = 0 .. nbins-1, so that sum_kappa
 * out[kappa] = mean of 1/2 rho |u|^2 over the plane.  out: HOST, nbins = ark_ke_spectrum_bins(nx, ny) doubles.  3D grids
 * with nz >= 8 (the scratch lives in the library's staging field, which ark_set/get_state_host also use).  Plain DFT with
 * fixed summation order (bit-reproducible).  Synchronises the stream.  Errors: ARK_EINVAL, ARK_ECUDA. */
int ark_ke_spectrum_bins(int nx, int ny);
int ark_ke_spectrum(ark_solver*, double* out, int nbins);

/* Ghost fill only, then copy the PADDED current state ((nx+4)*(ny+4)*(nz+4 or 1) per field, x fastest)
 * to device arrays: test hook for the boundary kernel.  Asynchronous. */
int ark_debug_get_padded(ark_solver*, double* rho, double* rhou, double* rhov, double* rhow, double* E);

/* Measurement hook: when enabled, every launch of the fused step kernel is bracketed by CUDA events on the
 * solver's stream (up to 4096 launches are kept; older ones are dropped).  ark_step_kernel_time() synchronises
 * the stream and returns the summed device time in milliseconds and the number of launches measured since
 * the last ark_step_kernel_timing(.., 1) call. */
int ark_step_kernel_timing(ark_solver*, int enable);
int ark_step_kernel_time(ark_solver*, double* total_ms, int* launches);

/* Measurement support (no handle): runs a register-resident DFMA-chain kernel on the current device and returns the
 * sustained fp64 instruction rate in 1e12 thread-instructions per second (one DFMA = one instruction).  bench.py
 * reports the "alu" roofline of the fp64-bound step kernel against it (the fp64 peak must be measured,
 * not derived).  Synchronises the stream. */
int ark_measure_fp64_peak(double* tinstr_per_s, void* cuda_stream);

/* Number of kernels this library has launched on behalf of the handle since creation. */
long long ark_launch_count(const ark_solver*);

void ark_destroy(ark_solver*);
const char* ark_last_error(void);
const char* ark_version_string(void);

#ifdef __cplusplus
}
#endif
#endif /* ARK_H */
