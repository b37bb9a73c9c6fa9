// ark_device.cuh -- device-side data layout and kernels of the ARK hot path (sm_100a).
//
// Scheme: PAPER.md (arXiv 1903.09043) sections 2.1-2.2 with readings A1..A20 of DESIGN.md.
// This file shares nothing with oracle/: every formula is restated here from the paper.
//
// HBM layout: SoA fp64, one padded array per conserved field (rho, rho*u, rho*v, [rho*w], E),
// 2 ghost layers per side (A9), x fastest, row pitch px (multiple of 16 doubles = 128 B).  Interior cell
// i = 0 sits at x index ARK_XOFF = 4 of a row (2 unused doubles, then the 2 low ghosts), so that the
// 28-wide output rows of the step kernel (tile origin a multiple of 28 = 7 sectors) start on a 32-byte
// sector boundary and every store of the hot kernel writes whole sectors.
#pragma once

#ifndef ARK_HOST_EMU
#include <cuda.h>           // CUtensorMap (type only; the encoder is fetched through the runtime, see ark.cu)
#include <cuda_runtime.h>
#define ARK_DEV __device__ __forceinline__
#define ARK_HD __host__ __device__
#define ARK_GLOBAL __global__
#define ARK_SHARED __shared__
#define ARK_DYN_SMEM(name) extern __shared__ double name[]
#else
// host emulation (tests only): the including translation unit supplies threadIdx & co, __syncthreads, rsqrt and the
// ARK_* macros BEFORE this header (tests/emu/ark_emu.h); nothing of it is part of the product build
#define ARK_HD
#endif

#define ARK_K_IMPEDANCE 1.1  // a = K max(rho_L c_L, rho_R c_R), reading A2
#define ARK_NG 2             // ghost layers (A9)
#define ARK_XOFF 4           // x index of interior cell 0 inside a padded row (>= ARK_NG)
#define ARK_MAX_ZCHUNKS 16   // z chunks of the 3D step kernel (blocks per column)

enum { ARK_BCK_PERIODIC = 0, ARK_BCK_REFLECTING = 1, ARK_BCK_FIXED_T = 2, ARK_BCK_FLUX = 3, ARK_BCK_EXTERNAL = 4 };

// Coefficients of the dissipative face flux (see ark_visc_face in ark_step.cuh).
struct ArkViscCoef { double cn, ct, c43, c23t, kh; };

// Constants derived from the parameters on the host (ark_fill_derived).  They travel with ArkParams in the kernel
// parameter (constant) bank, where fp64 instructions read them as operands: nothing uniform occupies a register.
struct ArkDerived {
    double inv_h, gh[3], dcoef;   // 1/h ; g_d h ; 2 ndim max(4 mu/3, (gamma-1) kappa) / h^2 (reading A4)
    int g_on[3];
    ArkViscCoef KV;
};

struct ArkParams {
    int nx, ny, nz, ndim, nf;   // interior sizes; nf = 4 (2D) or 5 (3D) stored fields
    int px, py, pz;             // padded extents (px is the row pitch)
    int offz;                   // 2 in 3D, 0 in 2D
    long long fstride;          // doubles between consecutive fields
    double h, gamma, gm1, g[3], mu, kappa;
    int theta;                  // 0: theta == 1 ; 1: eq. (13)
    int bc[3][2];
    double bcv[3][2];
    ArkDerived D;
    // general path: energy form (0: rho*E with the gravity work of PAPER.md:204-208;
    // 1: the non-conservative scheme of Appendix B) and an optional array-valued potential
    // (PAPER.md:55, :152), padded like a state field with its ghost values already filled (reading A25); NULL = -g.x
    int eform;
    const double* phi;
    // 3D step kernel: planes [zb[c], zb[c+1]) of z chunk c = blockIdx.z (chunk sizes decrease so that the last wave of
    // blocks is short; chosen by a scheduling simulation in ark_create)
    int zb[ARK_MAX_ZCHUNKS + 1];
};

inline void ark_fill_derived(ArkParams& P) {
    ArkDerived& D = P.D;
    D.inv_h = 1.0 / P.h;
    for (int d = 0; d < 3; ++d) { D.gh[d] = P.g[d] * P.h; D.g_on[d] = D.gh[d] != 0.0; }
    const double a = 4.0 * P.mu / 3.0, b = P.gm1 * P.kappa;
    D.dcoef = 2.0 * P.ndim * (a > b ? a : b) * D.inv_h * D.inv_h;
    D.KV.cn = P.mu * D.inv_h; D.KV.ct = 0.25 * P.mu * D.inv_h; D.KV.c43 = (4.0 / 3.0) * P.mu * D.inv_h;
    D.KV.c23t = (2.0 / 3.0) * 0.25 * P.mu * D.inv_h; D.KV.kh = P.kappa * D.inv_h;
}

// padded linear index of interior-based cell (i,j,k); ghosts are -2,-1 and n,n+1
ARK_DEV long long ark_idx(const ArkParams& P, int i, int j, int k) {
    return (long long)(i + ARK_XOFF) + (long long)P.px * ((long long)(j + ARK_NG) + (long long)P.py * (long long)(k + P.offz));
}

// NaN-propagating max (fmax would drop NaNs): SURVEY 8(a) row 8
ARK_DEV double ark_nanmax(double a, double b) { return (a != a) ? a : ((b != b) ? b : (a > b ? a : b)); }

// The same for values that are >= 0 when valid (CFL rates), on the integer pipe: for non-negative doubles the
// IEEE-754 bit pattern is monotone as an unsigned integer, every NaN and every negative value compares above
// +inf, so an unsigned max keeps the largest rate and lets any invalid value win (it is then reported as
// non-finite / non-positive by the caller).  Keeps DSETP traffic off the fp64 pipe in the step kernel.
typedef unsigned long long ark_u64;
ARK_DEV ark_u64 ark_rate_bits(double r) { return (ark_u64)__double_as_longlong(r); }
ARK_DEV double ark_rate_from_bits(ark_u64 b) { return __longlong_as_double((long long)b); }
ARK_DEV ark_u64 ark_umax(ark_u64 a, ark_u64 b) { return a > b ? a : b; }

// ------------------------------------------------------------------------------------------------
// Fast fp64 reciprocal and reciprocal square root for the step kernel: the hardware seed (MUFU.RCP64H /
// MUFU.RSQ64H through rcp/rsqrt.approx.ftz.f64; measured on B200: relative error 9.8e-7 / 9.1e-7) followed by ONE
// third-order Newton step, no special-case branches (arguments are finite, normal and positive for every valid cell;
// garbage lanes may produce inf/NaN that no valid cell consumes).  Measured maximum relative error over 2^20 random
// arguments in [2^-20, 2^21): 1.11e-16 (rcp), 1.38e-16 (rsqrt), i.e. <= 1.25 x 2^-53 -- against ~10 fp64
// instructions plus a slow-path call for the IEEE division.
// ------------------------------------------------------------------------------------------------
// ARK_STRICT (libark_b200_strict.so, built with --fmad=false): IEEE division and square root instead, so that the
// kernels' arithmetic differs from a plain evaluation only in what the source itself reorders (reading A20 on hardware).
#if defined(ARK_HOST_EMU) || defined(ARK_STRICT)
#define ARK_IEEE_RCP 1
#endif
ARK_DEV double ark_rcp(double x) {
#ifndef ARK_IEEE_RCP
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    e = fma(e, e, e);
    return fma(y, e, y);               // y (1 + e + e^2): error ~ seed^3
#else
    return 1.0 / x;
#endif
}

ARK_DEV double ark_rsqrt(double x) {
#ifndef ARK_IEEE_RCP
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);              // 1 - x y^2
    return fma(y * e, fma(0.375, e, 0.5), y);          // y (1 + e/2 + 3 e^2/8): error ~ seed^3
#else
    return 1.0 / sqrt(x);
#endif
}

// TMA tile loads global -> shared (cp.async.bulk.tensor, SASS UTMALDG) completing on an mbarrier: the U^n prefetch
// ring of the 3D step kernel.  ONE thread of the block issues ONE instruction per plane: a 4-D box (RX columns x RY rows
// x 1 plane x 5 fields) of the padded SoA state; out-of-range columns / rows of ragged tiles are zero-filled by the TMA
// unit.  The data never passes through registers or the LSU pipe.  (Host emulation: see ark_step.cuh, the copies are
// done synchronously per thread.)
#ifndef ARK_HOST_EMU
ARK_DEV unsigned ark_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
ARK_DEV void ark_mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ark_smem_u32(bar)), "r"(count) : "memory");
}
ARK_DEV void ark_mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
ARK_DEV void ark_mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ark_smem_u32(bar)), "r"(bytes) : "memory");
}
ARK_DEV void ark_tma_load_4d(double* smem_dst, const void* tmap, int c0, int c1, int c2, int c3, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(ark_smem_u32(smem_dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(ark_smem_u32(bar)) : "memory");
}
ARK_DEV void ark_mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "ARK_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra ARK_DONE_%=;\n"
        "bra ARK_WAIT_%=;\n"
        "ARK_DONE_%=:\n"
        "}\n" ::"r"(ark_smem_u32(bar)), "r"(parity) : "memory");
}
#endif

// ------------------------------------------------------------------------------------------------
// Tensor memory (TMEM, 256 KB per SM) as a per-thread scratch space.  The step kernel has no tensor-core work, so
// the whole TMEM of the SM is free: a warp may address lanes 32*(warp%4) .. +31, i.e. thread `lane` of a warp owns
// one TMEM lane, and the 512 32-bit columns of that lane are split among the warps that share the lane quarter.
// tcgen05.st / tcgen05.ld (shape 32x32b: one column = one 32-bit word per thread) move registers <-> TMEM on a
// datapath of their own (measured on B200: > 460 B/clk/SM with 8 warps, ~30 cycles load-to-use), which relieves both
// the register file (the z pipeline of a column is parked there between its uses) and the shared-memory pipe.
// A double occupies two adjacent columns.  ark_tm_ld must be followed by ark_tm_wait_ld() before the values are
// used; ark_tm_wait_st() orders earlier stores before later loads of the same columns.
// ------------------------------------------------------------------------------------------------
#ifndef ARK_HOST_EMU
// The "memory" clobber makes every TMEM transfer a scheduling fence for shared / global accesses (TMEM is not memory the
// compiler knows about: the volatile asm statements keep their own relative order)
#define ARK_TM_CLOBBER "memory"
#define ARK_LO(x) "r"(__double2loint(x))
#define ARK_HI(x) "r"(__double2hiint(x))
ARK_DEV unsigned ark_tm_alloc_all(unsigned* slot_in_smem) {           // one full warp; 512 columns = the whole TMEM
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(ark_smem_u32(slot_in_smem)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    return 0;
}
ARK_DEV void ark_tm_free_all(unsigned base) {                         // the same warp that allocated
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}
ARK_DEV void ark_tm_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
ARK_DEV void ark_tm_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
ARK_DEV void ark_tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
ARK_DEV void ark_tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
ARK_DEV void ark_tm_st1(unsigned a, double v0) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(a), ARK_LO(v0), ARK_HI(v0) : ARK_TM_CLOBBER);
}
ARK_DEV void ark_tm_st2(unsigned a, double v0, double v1) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), ARK_LO(v0), ARK_HI(v0), ARK_LO(v1), ARK_HI(v1) : ARK_TM_CLOBBER);
}
ARK_DEV void ark_tm_ld2(unsigned a, double& v0, double& v1) {
    int l0, h0, l1, h1;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(l0), "=r"(h0), "=r"(l1), "=r"(h1) : "r"(a) : ARK_TM_CLOBBER);
    v0 = __hiloint2double(h0, l0); v1 = __hiloint2double(h1, l1);
}
// Wider groups go as single-double transfers: x8 / x16 tcgen05 shapes need their 8 / 16 registers contiguous, and the
// register-packing moves that costs were measured to outweigh the saved instructions (profiles/r02_step_kernel.md).
ARK_DEV void ark_tm_st4(unsigned a, double v0, double v1, double v2, double v3) { ark_tm_st1(a, v0); ark_tm_st1(a + 2, v1); ark_tm_st1(a + 4, v2); ark_tm_st1(a + 6, v3); }
ARK_DEV void ark_tm_st8(unsigned a, double v0, double v1, double v2, double v3, double v4, double v5, double v6, double v7) {
    ark_tm_st4(a, v0, v1, v2, v3); ark_tm_st4(a + 8, v4, v5, v6, v7);
}
ARK_DEV void ark_tm_ld1(unsigned a, double& v0) {
    int l0, h0;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(l0), "=r"(h0) : "r"(a) : ARK_TM_CLOBBER);
    v0 = __hiloint2double(h0, l0);
}
ARK_DEV void ark_tm_ld4(unsigned a, double& v0, double& v1, double& v2, double& v3) { ark_tm_ld1(a, v0); ark_tm_ld1(a + 2, v1); ark_tm_ld1(a + 4, v2); ark_tm_ld1(a + 6, v3); }
ARK_DEV void ark_tm_ld8(unsigned a, double& v0, double& v1, double& v2, double& v3, double& v4, double& v5, double& v6, double& v7) {
    ark_tm_ld4(a, v0, v1, v2, v3); ark_tm_ld4(a + 8, v4, v5, v6, v7);
}
#endif

// ------------------------------------------------------------------------------------------------
// Primitive variables of one cell (PAPER.md:315-319 ideal gas, c^2 = gamma p / rho; :370 p = rho T).
// rc = rho*c and irc = 1/(rho*c) come from ONE rsqrt: rho*c = sqrt(gamma p rho).
// ------------------------------------------------------------------------------------------------
struct ArkPrim { double rho, u, v, w, p, rc, irc, T; };

ARK_DEV ArkPrim ark_prim(const ArkParams& P, double rho, double mx, double my, double mz, double E) {
    ArkPrim q;
    const double rinv = 1.0 / rho;
    q.rho = rho;
    q.u = mx * rinv;
    q.v = my * rinv;
    q.w = mz * rinv;
    const double ke = 0.5 * (mx * q.u + my * q.v + mz * q.w);
    q.p = P.gm1 * (E - ke);
    const double gpr = P.gamma * q.p * rho;        // (rho c)^2
#ifdef ARK_STRICT
    q.irc = 1.0 / sqrt(gpr);
#else
    q.irc = rsqrt(gpr);
#endif
    q.rc = gpr * q.irc;
    q.T = q.p * rinv;
    return q;
}

// The same with ark_rcp / ark_rsqrt (step kernel only; the ghost fill keeps the IEEE version above).
ARK_DEV ArkPrim ark_prim_fast(const ArkParams& P, double rho, double mx, double my, double mz, double E) {
    // arranged for a short dependency chain: |m|^2 and gamma (gamma-1) rho do not wait for the reciprocal
    ArkPrim q;
    const double hm2 = 0.5 * (mx * mx + my * my + mz * mz);
    const double ggr = (P.gamma * P.gm1) * rho;
    const double rinv = ark_rcp(rho);
    q.rho = rho;
    q.u = mx * rinv;
    q.v = my * rinv;
    q.w = mz * rinv;
    const double ei = E - hm2 * rinv;              // rho e
    q.p = P.gm1 * ei;
    const double gpr = ggr * ei;                   // (rho c)^2 = gamma p rho
    q.irc = ark_rsqrt(gpr);
    q.rc = gpr * q.irc;
    q.T = q.p * rinv;
    return q;
}

// ------------------------------------------------------------------------------------------------
// Acoustic face between L and R along one axis (PAPER.md:152 for a, S, u*, Pi*; PAPER.md:218-222
// for theta, eq. 13).  un = face-normal velocity, gh = g_d * h (Phi_R - Phi_L = -g_d h, A12).
// Divisions by a and by max(c_L,c_R) are replaced by min() of the per-cell reciprocals:
//   1/(2a) = min(irc_L, irc_R)/(2K),  1/max(c_L,c_R) = min(rho_L irc_L, rho_R irc_R).
// ------------------------------------------------------------------------------------------------
struct ArkFace { double us, pi, S; };

ARK_DEV ArkFace ark_face(int theta_on, double gh,
                         double rhoL, double unL, double pL, double rcL, double ircL,
                         double rhoR, double unR, double pR, double rcR, double ircR) {
    ArkFace f;
    // one comparison picks max(rc) and min(1/rc) (plain selects: fmax/fmin on doubles cost ~6 instructions)
    const bool lg = rcL > rcR;
    const double a = ARK_K_IMPEDANCE * (lg ? rcL : rcR);
    const double i2a = (0.5 / ARK_K_IMPEDANCE) * (lg ? ircL : ircR);
    f.S = (0.5 * gh) * (rhoL + rhoR);
    f.us = 0.5 * (unL + unR) - ((pR - pL) - f.S) * i2a;
    double ath = a;
    if (theta_on) {
        const double icL = rhoL * ircL, icR = rhoR * ircR;          // 1/c
        const double ma = fabs(f.us) * (icL < icR ? icL : icR);     // |u*| / max(c_L, c_R)
        ath = a * (ma < 1.0 ? ma : 1.0);
    }
    f.pi = 0.5 * (pL + pR) - 0.5 * ath * (unR - unL);
    return f;
}

// ------------------------------------------------------------------------------------------------
// dense <-> padded copies
// ------------------------------------------------------------------------------------------------
ARK_GLOBAL void ark_k_pack(ArkParams P, double* __restrict__ U, const double* __restrict__ src, int field) {
    const long long n = (long long)P.nx * P.ny * P.nz;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(s % P.nx);
        const long long r = s / P.nx;
        const int j = (int)(r % P.ny), k = (int)(r / P.ny);
        U[field * P.fstride + ark_idx(P, i, j, k)] = src[s];
    }
}

ARK_GLOBAL void ark_k_unpack(ArkParams P, const double* __restrict__ U, double* __restrict__ dst, int field) {
    const long long n = (long long)P.nx * P.ny * P.nz;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(s % P.nx);
        const long long r = s / P.nx;
        const int j = (int)(r % P.ny), k = (int)(r / P.ny);
        dst[s] = U[field * P.fstride + ark_idx(P, i, j, k)];
    }
}

// padded (pitch px) -> padded dense (pitch nx+4): debug / test hook for the ghost fill
ARK_GLOBAL void ark_k_unpack_padded(ArkParams P, const double* __restrict__ U, double* __restrict__ dst, int field) {
    const int mx = P.nx + 2 * ARK_NG;
    const long long n = (long long)mx * P.py * P.pz;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(s % mx);
        const long long r = s / mx;
        dst[s] = U[field * P.fstride + (long long)(i + ARK_XOFF - ARK_NG) + (long long)P.px * r];
    }
}

// ------------------------------------------------------------------------------------------------
// Ghost fill along one axis (A9).  Launched for AXIS = 0, 1, 2 in this order; each later axis sweeps
// the already-extended range of the earlier ones, so edges and corners are filled.  One thread per
// (transverse position, side); it writes ghost layers 1 then 2 (layer 2 chains eq. (14) from layer 1).
//   periodic: copy.   reflecting wall: u_n -> -u_n, T_g = T_src.
//   fixed-T no-slip wall: u -> -u (all components), T_g = 2 T_w - T_src.
//   imposed-flux wall (A22): u_n -> -u_n, T_g = T_src + (2l-1) F h / kappa (F = heat flux entering).
//   external (ghost zones that hold the neighbouring sub-domain's cells): left as the caller set them.
//   rho_g from the discrete hydrostatic relation (14), PAPER.md:237:
//       p_g - p_prev = 1/2 (rho_prev + rho_g) delta,  delta = Phi_prev - Phi_g = -+ g_d h,  p_g = rho_g T_g
//       (with an array-valued potential, P.phi: the difference of its padded values).
// ------------------------------------------------------------------------------------------------
template <int AXIS>
ARK_GLOBAL void ark_k_bc(ArkParams P, double* __restrict__ U) {
    // transverse extents (a = faster transverse axis, b = slower one)
    int na, nb, loa, lob;
    if (AXIS == 0)      { na = P.ny;            loa = 0;        nb = P.nz;                        lob = 0; }
    else if (AXIS == 1) { na = P.nx + 2 * ARK_NG; loa = -ARK_NG; nb = P.nz;                        lob = 0; }
    else                { na = P.nx + 2 * ARK_NG; loa = -ARK_NG; nb = P.ny + 2 * ARK_NG;           lob = -ARK_NG; }
    const long long ntr = (long long)na * nb;
    const int n = AXIS == 0 ? P.nx : (AXIS == 1 ? P.ny : P.nz);
    const long long sd = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)P.px : (long long)P.px * P.py);
    const double* __restrict__ Uc = U;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < 2 * ntr; s += (long long)gridDim.x * blockDim.x) {
        const int side = (int)(s / ntr);
        const long long r = s % ntr;
        const int a = loa + (int)(r % na), b = lob + (int)(r / na);
        int c[3];
        if (AXIS == 0)      { c[0] = 0; c[1] = a; c[2] = b; }
        else if (AXIS == 1) { c[0] = a; c[1] = 0; c[2] = b; }
        else                { c[0] = a; c[1] = b; c[2] = 0; }
        const long long base = ark_idx(P, c[0], c[1], c[2]);     // index of interior cell 0 along AXIS
        const int type = P.bc[AXIS][side];
        if (type == ARK_BCK_EXTERNAL) continue;                   // ghost planes supplied by the caller (slab decomposition, ark_set_halo)
        for (int l = 1; l <= ARK_NG; ++l) {
            const int ig = side == 0 ? -l : n - 1 + l;
            const long long jg = base + ig * sd;
            if (type == ARK_BCK_PERIODIC) {
                const int is = side == 0 ? n - l : l - 1;
                const long long js = base + is * sd;
                for (int f = 0; f < P.nf; ++f) U[f * P.fstride + jg] = Uc[f * P.fstride + js];
                continue;
            }
            const int is = side == 0 ? l - 1 : n - l;             // mirror cell
            const int ip = side == 0 ? ig + 1 : ig - 1;           // previous cell of the hydrostatic chain
            const long long js = base + is * sd, jp = base + ip * sd;
            const long long fE = (long long)(P.nf - 1) * P.fstride;
            const double mzs = P.ndim == 3 ? U[3 * P.fstride + js] : 0.0;
            const double mzp = P.ndim == 3 ? U[3 * P.fstride + jp] : 0.0;
            const ArkPrim ws = ark_prim(P, U[js], U[P.fstride + js], U[2 * P.fstride + js], mzs, U[fE + js]);
            const ArkPrim wp = ark_prim(P, U[jp], U[P.fstride + jp], U[2 * P.fstride + jp], mzp, U[fE + jp]);
            double ug[3] = {ws.u, ws.v, ws.w};
            double Tg;
            if (type == ARK_BCK_REFLECTING) {
                ug[AXIS] = -ug[AXIS];
                Tg = ws.T;
            } else if (type == ARK_BCK_FLUX) {
                ug[AXIS] = -ug[AXIS];
                Tg = ws.T + (2 * l - 1) * P.bcv[AXIS][side] * P.h / P.kappa;
            } else {
                ug[0] = -ug[0]; ug[1] = -ug[1]; ug[2] = -ug[2];
                Tg = 2.0 * P.bcv[AXIS][side] - ws.T;
            }
            const double delta = P.phi ? P.phi[jp] - P.phi[jg] : (side == 0 ? -1.0 : 1.0) * P.g[AXIS] * P.h;
            double rg = (wp.p + 0.5 * wp.rho * delta) / (Tg - 0.5 * delta);
            // A9 needs T_g > |g_d| h / 2: otherwise relation (14) has no positive solution; flag the cell (NaN reaches the
            // CFL reduction, which reports ARK_ENONFINITE) instead of marching on with a negative ghost density
            // (only ghost cells that face interior cells: edge / corner ghosts mirror ghost cells of another wall and only
            // their velocity is ever used, by the diagonal points of the viscous stencil)
            const bool faces_interior = (AXIS == 0) || (c[0] >= 0 && c[0] < P.nx && (AXIS == 1 || (c[1] >= 0 && c[1] < P.ny)));
            if (faces_interior && !(rg > 0.0)) rg = __longlong_as_double(0x7ff8000000000000LL);
            const double pg = rg * Tg;
            U[jg] = rg;
            U[P.fstride + jg] = rg * ug[0];
            U[2 * P.fstride + jg] = rg * ug[1];
            if (P.ndim == 3) U[3 * P.fstride + jg] = rg * ug[2];
            U[fE + jg] = pg / P.gm1 + 0.5 * rg * (ug[0] * ug[0] + ug[1] * ug[1] + ug[2] * ug[2]);
        }
    }
}

// Periodic x sweep: a pure copy of two cells per (row, side, field).  The general kernel above walks the fields and
// layers of a row end serially in one thread; every access of this sweep is a lone 32-byte sector (row ends are a
// pitch apart), so the only lever is parallelism: one thread per (row, side, field), both layers in one 16-byte
// access when nx is even (ghost and source pairs are then 16-byte aligned: interior cell 0 sits at an even index).
ARK_GLOBAL void ark_k_bc_x_periodic(ArkParams P, double* __restrict__ U) {
    const long long nrow = (long long)P.ny * P.nz;
    const long long n = nrow * 2 * P.nf;
    const bool vec = (P.nx & 1) == 0;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int f = (int)(s / (2 * nrow));
        const long long rem = s - (long long)f * 2 * nrow;
        const int side = (int)(rem / nrow);
        const long long r = rem - (long long)side * nrow;
        const long long base = f * P.fstride + ark_idx(P, 0, (int)(r % P.ny), (int)(r / P.ny));
        const long long dst = side == 0 ? base - ARK_NG : base + P.nx;            // ghosts -2,-1 | nx,nx+1
        const long long src = side == 0 ? base + P.nx - ARK_NG : base;            // cells nx-2,nx-1 | 0,1
#ifndef ARK_HOST_EMU
        if (vec) { *reinterpret_cast<double2*>(U + dst) = *reinterpret_cast<const double2*>(U + src); continue; }
#endif
        const double a = U[src], b = U[src + 1];
        U[dst] = a; U[dst + 1] = b;
        (void)vec;
    }
}

// Ghost values of an array-valued potential (reading A25): periodic axes wrap, wall axes continue Phi
// linearly from the two cells next to the wall (Phi(-l) = Phi(0) + l (Phi(0) - Phi(1))), which reproduces a constant
// gravity exactly.  Same x, y, z sweep order over the already-extended ranges as the state's ghost fill; runs once, in
// ark_set_potential.  One thread per (transverse position).
template <int AXIS>
ARK_GLOBAL void ark_k_phi_ghosts(ArkParams P, double* __restrict__ phi) {
    int na, nb, loa, lob;
    if (AXIS == 0)      { na = P.ny;            loa = 0;        nb = P.nz;                        lob = 0; }
    else if (AXIS == 1) { na = P.nx + 2 * ARK_NG; loa = -ARK_NG; nb = P.nz;                        lob = 0; }
    else                { na = P.nx + 2 * ARK_NG; loa = -ARK_NG; nb = P.ny + 2 * ARK_NG;           lob = -ARK_NG; }
    const long long ntr = (long long)na * nb;
    const int n = AXIS == 0 ? P.nx : (AXIS == 1 ? P.ny : P.nz);
    const long long sd = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)P.px : (long long)P.px * P.py);
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < ntr; r += (long long)gridDim.x * blockDim.x) {
        const int a = loa + (int)(r % na), b = lob + (int)(r / na);
        const long long base = AXIS == 0 ? ark_idx(P, 0, a, b) : (AXIS == 1 ? ark_idx(P, a, 0, b) : ark_idx(P, a, b, 0));
        for (int l = 1; l <= ARK_NG; ++l) {
            if (P.bc[AXIS][0] == ARK_BCK_PERIODIC) {
                phi[base - l * sd] = phi[base + (n - l) * sd];
                phi[base + (n - 1 + l) * sd] = phi[base + (l - 1) * sd];
            } else {
                const double p0 = phi[base], p1 = phi[base + sd], q0 = phi[base + (n - 1) * sd], q1 = phi[base + (n - 2) * sd];
                phi[base - l * sd] = p0 + l * (p0 - p1);
                phi[base + (n - 1 + l) * sd] = q0 + l * (q0 - q1);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// CFL rate of one cell (reading A4):
//   rate = sum_d (|u_d| + c)/h + 2 ndim max(4 mu/3, (gamma-1) kappa) / (rho h^2)
// ------------------------------------------------------------------------------------------------
ARK_DEV double ark_rate(const ArkParams& P, double rho, double mx, double my, double mz, double E,
                        double inv_h, double dcoef) {
    const double rinv = 1.0 / rho;
    const double u = mx * rinv, v = my * rinv, w = mz * rinv;
    const double p = P.gm1 * (E - 0.5 * (mx * u + my * v + mz * w));
    const double c = sqrt(P.gamma * p * rinv);
    const double s = fabs(u) + fabs(v) + (P.ndim == 3 ? fabs(w) : 0.0) + (double)P.ndim * c;
    return s * inv_h + dcoef * rinv;
}

// block-wide NaN-propagating max: warp shuffles, then one value per warp through shared memory.
// Every thread of the block must call it; the result is valid in thread 0.
ARK_DEV double ark_block_nanmax(double v, double* red /* >= 32 doubles of shared memory */) {
#ifndef ARK_HOST_EMU
    for (int o = 16; o > 0; o >>= 1) v = ark_nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = lane < nw ? red[lane] : -1.0;
        for (int o = 16; o > 0; o >>= 1) v = ark_nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    }
#else
    v = ark_emu_block_nanmax(v);
#endif
    return v;
}

// pass 1: grid-stride running max per thread -> one value per block in scratch[blockIdx.x]
ARK_GLOBAL void ark_k_cfl_pass1(ArkParams P, const double* __restrict__ U, double* __restrict__ scratch) {
    ARK_SHARED double red[32];
    const long long n = (long long)P.nx * P.ny * P.nz;
    const double inv_h = 1.0 / P.h;
    const double dcoef = 2.0 * P.ndim * fmax(4.0 * P.mu / 3.0, P.gm1 * P.kappa) * inv_h * inv_h;
    const long long fE = (long long)(P.nf - 1) * P.fstride;
    double m = -1.0;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(s % P.nx);
        const long long r = s / P.nx;
        const long long c = ark_idx(P, i, (int)(r % P.ny), (int)(r / P.ny));
        const double mz = P.ndim == 3 ? U[3 * P.fstride + c] : 0.0;
        m = ark_nanmax(m, ark_rate(P, U[c], U[P.fstride + c], U[2 * P.fstride + c], mz, U[fE + c], inv_h, dcoef));
    }
    m = ark_block_nanmax(m, red);
    if (threadIdx.x == 0) scratch[blockIdx.x] = m;
}

// ------------------------------------------------------------------------------------------------
// Diagnostics the paper reports (PAPER.md:398-407 maximum velocity, :435 mean absolute velocity, :14 conserved mass
// and total energy): max |u|, sum |u|, sum 1/2 rho |u|^2, max Mach, sum rho, sum (E + rho Phi), Phi = -g.x at the
// cell centres.  Two passes without atomics: fixed grid-stride order per thread, fixed shuffle tree per block, one
// block over the per-block partials -- the result is bit-reproducible for a given grid.
// ------------------------------------------------------------------------------------------------
#define ARK_NDIAG 6
ARK_DEV void ark_diag_combine(double* a, const double* b) {
    a[0] = ark_nanmax(a[0], b[0]); a[1] += b[1]; a[2] += b[2]; a[3] = ark_nanmax(a[3], b[3]); a[4] += b[4]; a[5] += b[5];
}
ARK_DEV void ark_diag_block(double* v, double* red /* 32 * ARK_NDIAG doubles of shared memory */) {
#ifndef ARK_HOST_EMU
    double o[ARK_NDIAG];
    for (int d = 16; d > 0; d >>= 1) {
        for (int f = 0; f < ARK_NDIAG; ++f) o[f] = __shfl_down_sync(0xffffffffu, v[f], d);
        ark_diag_combine(v, o);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) for (int f = 0; f < ARK_NDIAG; ++f) red[wid * ARK_NDIAG + f] = v[f];
    __syncthreads();
    if (threadIdx.x == 0)
        for (int w2 = 1; w2 < nw; ++w2) ark_diag_combine(v, red + w2 * ARK_NDIAG);
#else
    (void)v; (void)red;
#endif
}
ARK_GLOBAL void ark_k_diag_pass1(ArkParams P, const double* __restrict__ U, double* __restrict__ part) {
    ARK_SHARED double red[32 * ARK_NDIAG];
    const long long n = (long long)P.nx * P.ny * P.nz;
    const long long fE = (long long)(P.nf - 1) * P.fstride;
    double v[ARK_NDIAG] = {0, 0, 0, 0, 0, 0};
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(s % P.nx);
        const long long r = s / P.nx;
        const int j = (int)(r % P.ny), k = (int)(r / P.ny);
        const long long c = ark_idx(P, i, j, k);
        const double rho = U[c], mx = U[P.fstride + c], my = U[2 * P.fstride + c], mz = P.ndim == 3 ? U[3 * P.fstride + c] : 0.0;
        const double E = U[fE + c];
        const double rinv = 1.0 / rho;
        const double m2 = mx * mx + my * my + mz * mz;
        const double ke = 0.5 * m2 * rinv;
        const double speed = sqrt(m2) * rinv;
        const double cs = sqrt(P.gamma * P.gm1 * (E - ke) * rinv);
        const double phi = P.phi ? P.phi[c] : -((i + 0.5) * P.g[0] + (j + 0.5) * P.g[1] + (P.ndim == 3 ? (k + 0.5) * P.g[2] : 0.0)) * P.h;
        const double w[ARK_NDIAG] = {speed, speed, ke, speed / cs, rho, E + rho * phi};
        ark_diag_combine(v, w);
    }
    ark_diag_block(v, red);
    if (threadIdx.x == 0) for (int f = 0; f < ARK_NDIAG; ++f) part[(long long)blockIdx.x * ARK_NDIAG + f] = v[f];
}
ARK_GLOBAL void ark_k_diag_pass2(const double* __restrict__ part, int nblocks, double* __restrict__ out) {
    ARK_SHARED double red[32 * ARK_NDIAG];
    double v[ARK_NDIAG] = {0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) ark_diag_combine(v, part + (long long)b * ARK_NDIAG);
    ark_diag_block(v, red);
    if (threadIdx.x == 0) for (int f = 0; f < ARK_NDIAG; ++f) out[f] = v[f];
}

// pass 2: single block over the per-block values; result[0] = max rate,
// result[1] = dt = cfl / max rate (used by the device-side time loop of ark_run).  With dt_log the step size is also
// appended at dt_log[*log_count] (a device-side counter, so that the launch can be replayed from a CUDA graph).
// result[3] is a STICKY flag (never cleared here): set to 1.0 when a maximum rate was not finite and positive, so that a
// device-side time loop (ark_run) can report a blown-up state without a host round trip per step (reading A15).
ARK_GLOBAL void ark_k_cfl_pass2(const double* __restrict__ scratch, int nvals, double cfl, double* __restrict__ result,
                                double* __restrict__ dt_log, int* __restrict__ log_count) {
    ARK_SHARED double red[32];
    double m = -1.0;
    for (int s = threadIdx.x; s < nvals; s += blockDim.x) m = ark_nanmax(m, scratch[s]);
    m = ark_block_nanmax(m, red);
    if (threadIdx.x == 0) {
        result[0] = m;
        result[1] = cfl / m;
        if (!(m > 0.0) || m > 1.7e308) result[3] = 1.0;
        if (dt_log) { const int i = *log_count; dt_log[i] = cfl / m; *log_count = i + 1; }
    }
}

// ------------------------------------------------------------------------------------------------
// Kinetic-energy power spectrum of the horizontal middle plane (Fig. 11; the paper prints no formula:
// reading A26 of DESIGN.md).  Plane k = nz/2, w_c = sqrt(rho) u_c = m_c / sqrt(rho), c = x, y, z;
//   w^_c(kx,ky) = 1/(nx ny) sum_{i,j} w_c(i,j) exp(-2 pi i (kx i / nx + ky j / ny)),
//   E(kappa) = sum over (kx,ky) with floor(sqrt(kx~^2 + ky~^2) + 1/2) == kappa of 1/2 sum_c |w^_c|^2   (kx~, ky~ signed),
// so that sum_kappa E(kappa) = mean over the plane of 1/2 rho |u|^2 (Parseval).  A plain separable DFT with tabulated
// twiddles (exact index arithmetic (kx i) mod nx, sincospi): O(n^3) per plane, milliseconds at 512^2, every sum in a
// fixed order (bit-reproducible, no atomics).  Diagnostic, not part of the time step.
// ------------------------------------------------------------------------------------------------
#ifndef ARK_HOST_EMU
ARK_GLOBAL void ark_k_spec_twiddle(double* __restrict__ tw, int n) {       // tw[2t], tw[2t+1] = cos, sin (2 pi t / n)
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x) {
        double sn, cs;
        sincospi(2.0 * (double)t / (double)n, &sn, &cs);
        tw[2 * t] = cs; tw[2 * t + 1] = sn;
    }
}
// A[c][j][kx] = sum_i w_c(i,j) exp(-2 pi i kx i / nx)   (complex, interleaved), one thread per (j, kx)
ARK_GLOBAL void ark_k_spec_rows(ArkParams P, const double* __restrict__ U, int kplane, const double* __restrict__ twx, double* __restrict__ A) {
    const long long n = (long long)P.nx * P.ny;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(s % P.nx), j = (int)(s / P.nx);
        const double* row = U + ark_idx(P, 0, j, kplane);
        double re[3] = {0, 0, 0}, im[3] = {0, 0, 0};
        int t = 0;
        for (int i = 0; i < P.nx; ++i) {
            const double isr = 1.0 / sqrt(row[i]);
            const double cs = twx[2 * t], sn = twx[2 * t + 1];
            for (int c = 0; c < 3; ++c) {
                const double w = row[(c + 1) * P.fstride + i] * isr;
                re[c] += w * cs; im[c] -= w * sn;
            }
            t += kx; if (t >= P.nx) t -= P.nx;
        }
        for (int c = 0; c < 3; ++c) { A[2 * (c * n + s)] = re[c]; A[2 * (c * n + s) + 1] = im[c]; }
    }
}
// Pw[ky][kx] = 1/2 sum_c |sum_j A[c][j][kx] exp(-2 pi i ky j / ny)|^2 / (nx ny)^2, one thread per (ky, kx)
ARK_GLOBAL void ark_k_spec_cols(ArkParams P, const double* __restrict__ A, const double* __restrict__ twy, double* __restrict__ Pw) {
    const long long n = (long long)P.nx * P.ny;
    const double norm = 1.0 / ((double)n * (double)n);
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(s % P.nx), ky = (int)(s / P.nx);
        double pw = 0.0;
        for (int c = 0; c < 3; ++c) {
            double re = 0.0, im = 0.0;
            int t = 0;
            for (int j = 0; j < P.ny; ++j) {
                const double ar = A[2 * (c * n + (long long)j * P.nx + kx)], ai = A[2 * (c * n + (long long)j * P.nx + kx) + 1];
                const double cs = twy[2 * t], sn = twy[2 * t + 1];
                re += ar * cs + ai * sn;                   // (ar + i ai)(cs - i sn)
                im += ai * cs - ar * sn;
                t += ky; if (t >= P.ny) t -= P.ny;
            }
            pw += re * re + im * im;
        }
        Pw[s] = 0.5 * pw * norm;
    }
}
// E[kappa] = sum of Pw over the shell of kappa: one block per kappa, fixed order
ARK_GLOBAL void ark_k_spec_bins(ArkParams P, const double* __restrict__ Pw, double* __restrict__ E) {
    ARK_SHARED double red[256];
    const int kappa = blockIdx.x;
    const long long n = (long long)P.nx * P.ny;
    double acc = 0.0;
    for (long long s = threadIdx.x; s < n; s += blockDim.x) {
        int kx = (int)(s % P.nx), ky = (int)(s / P.nx);
        if (2 * kx > P.nx) kx -= P.nx;
        if (2 * ky > P.ny) ky -= P.ny;
        const int b = (int)floor(sqrt((double)(kx * kx + ky * ky)) + 0.5);
        if (b == kappa) acc += Pw[s];
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) E[kappa] = red[0];
}
#endif

// ------------------------------------------------------------------------------------------------
// fp64 pipe microbenchmark (measurement support for the "alu" roofline of bench.py): register-resident DFMA chains,
// 8 independent chains per thread, no memory traffic.  One DFMA = one fp64 instruction (SURVEY 8(d) asks for a
// MEASURED fp64 peak next to the measured HBM peak).
// ------------------------------------------------------------------------------------------------
ARK_GLOBAL void ark_k_dfma_peak(double* __restrict__ sink, int iters, double a, double b) {
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (r == 123.456) sink[0] = r;             // never true for the arguments used; keeps the chains alive
}

