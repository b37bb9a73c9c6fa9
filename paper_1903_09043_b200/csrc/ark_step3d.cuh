// ark_step3d.cuh -- the fused full-step kernel in 3D (acoustic + transport + dissipative + update + CFL epilogue).
//
// One launch advances U^n -> U^{n+1}: every conserved field is read once and written once (80 B per cell update);
// all face quantities, velocity gradients and the intermediate state U~ live in registers / shared memory only.
//
// Decomposition ("2.5-D marching", two rows per thread): a block owns a TX x TY tile of (x,y) columns plus a 2-cell
// halo (region RX x RY = (TX+4) x (TY+4), RX = 32 in the product build) and marches along z over a chunk of planes.
// A WARP OWNS TWO ADJACENT REGION ROWS (a, b = a+1): lane = x position, every thread carries the z pipelines of its
// two columns in registers.  What the two rows exchange (their common y face, the centred y differences, the
// upwind U~) never leaves the thread; x neighbours are reached by warp shuffles; only the row pair below / above is
// reached through shared memory.  Every face flux is computed ONCE (by the cell above / right of / behind the face)
// and handed to the other side, so the update is a difference of single-valued face fluxes (eq. 11).
//
// Row pairs m = 0 .. NW-1 of a block:  m = 0 : (edge row 0, ring row 1)  -- ROLE 0
//                                      m = 1 .. NW-2 : two tile rows     -- ROLE 1
//                                      m = NW-1 : (ring row RY-2, edge row RY-1) -- ROLE 2
// Edge rows only provide primitives, ring rows also faces and U~ (PAPER.md:158-160 needs all faces of a cell), tile
// rows are the outputs.  The role is a compile-time parameter of the whole plane loop and warp-uniform.
//
// Warp specialisation with register reallocation (setmaxnreg): the block has NW + 2 warps.  Warpgroup 0 (warps 0-3)
// holds the two light ring pairs (warp 0: ring row 1, warp 1: ring row RY-2; warps 2, 3 compute the primitives of the
// edge rows 0 and RY-1 for them) and shrinks its register allowance; the tile pairs run on warps 4 .. NW+1 and grow theirs, so that every scheduler of
// the SM (warp w issues on scheduler w % 4) carries the same number of heavy tile warps.  The z pipeline of a column
// (primitives of three planes, U~, running update, centred differences) is parked in TMEM between its uses.
//
// Per plane q one iteration does (2 block barriers):
//   S1  primitives of plane q+1 of the own two columns (from the TMA-filled U^n ring)
//   S2  acoustic faces: x- (left cell by shuffle), y- of row a (row a-1 from shared memory),
//       the face between a and b, z+ (q|q+1); centred velocity differences of plane q
//   --- barrier B
//   S3  acoustic update U~(q); z face (q-1|q): transport + dissipative flux, which completes
//       plane q-1 -> store U^{n+1}(q-1), CFL rate; x faces and the (a|b) face of plane q: transport (upwind on u*,
//       PAPER.md:170-174) + dissipative fluxes -> running update of plane q
//   --- barrier C
//   S4  low-y face of row a (U~ of row a-1 from shared memory): flux -> own update, and -> shared memory for the
//       pair below, which subtracts it when it completes that plane one iteration later.
#pragma once
#include "ark_step.cuh"

enum { ARK_ROW_EDGE = 0, ARK_ROW_RING = 1, ARK_ROW_TILE = 2 };
ARK_HD constexpr int ark_row_kind(int role, int r) {
    return role == 1 ? ARK_ROW_TILE : ((role == 0) == (r == 0) ? ARK_ROW_EDGE : ARK_ROW_RING);
}

// x-neighbour exchange: lane - 1 / lane + 1 of the warp (a region row is exactly one warp)
#ifndef ARK_HOST_EMU
ARK_DEV double ark_xl(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
ARK_DEV double ark_xr(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
#else
ARK_DEV double ark_xl(double v) { return ark_emu_shfl(v, -1); }
ARK_DEV double ark_xr(double v) { return ark_emu_shfl(v, +1); }
#endif

// TX outputs per row (RX = TX + 4 lanes), NW row pairs per block on NW + 2 warps.
template <bool VISC, int TX, int NW>
struct ArkCfg3 {
    static constexpr int RX = TX + 4, RY = 2 * NW, TY = RY - 4, NCOL = RX * RY;
    static constexpr int NS = RX * NW;          // exchange slots: one per (pair, lane)
    static constexpr int NWARP = NW + 2, NT = RX * NWARP;
    static constexpr int REG_RING = ARK_REG_RING, REG_TILE = ARK_REG_TILE;   // setmaxnreg targets of warpgroup 0 / the others
    static constexpr int NP = VISC ? 8 : 7;                          // rho,u,v,w,p,rc,irc(,T): T only feeds the heat flux
    // shared memory, in doubles.  UR is the TMA destination: offset 0, slot size a multiple of 128 B.
    static constexpr int UR_OFF = 0;                                 // [3][5][NCOL]  U^n of planes q, q+1, q+2
    static constexpr int PBB_OFF = UR_OFF + 15 * NCOL;               // [2][NP][NS]   primitives of row b, planes q, q+1
    static constexpr int PBA_OFF = PBB_OFF + 2 * NP * NS;            // [2][3][NS]    u,v,w of row a (VISC)
    static constexpr int FB_OFF = PBA_OFF + (VISC ? 6 : 0) * NS;     // [3][NS]       u*, Pi*, S of the low-y face of row a
    static constexpr int TB_OFF = FB_OFF + 3 * NS;                   // [5][NS]       U~ of row b
    static constexpr int YB_OFF = TB_OFF + 5 * NS;                   // [5][NS]       flux through the low-y face of row a
    static constexpr int GB_OFF = YB_OFF + 5 * NS;                   // [4][NS]       dxv,dxu,dzv,dzw of row b (VISC)
    static constexpr int EB_OFF = GB_OFF + (VISC ? 4 : 0) * NS;      // [2][2][5][RX]  rho,v,p,rc,irc of the two edge rows, planes q, q+1
    static constexpr int RED_OFF = EB_OFF + 20 * RX;                 // [32] block reduction of the rate
    static constexpr int MBAR_OFF = RED_OFF + 32;                    // [3] mbarriers of the UR slots, [3] TMEM base, [4] mbarrier of barrier B
    static constexpr int SMEM_DOUBLES = MBAR_OFF + 6;
    static constexpr size_t SMEM_BYTES = (size_t)SMEM_DOUBLES * sizeof(double);
    static_assert((5 * NCOL * sizeof(double)) % 128 == 0, "TMA destination slots must stay 128-byte aligned");
    static_assert(((NWARP + 3) / 4) * 144 <= 512, "TMEM scratch columns of the warps that share a lane quarter");
    static_assert(NWARP % 4 == 0 || RX != 32, "whole warpgroups (setmaxnreg)");
    // warp -> row pair: warp 0: pair 0 (low ring), warp 1: pair NW-1 (high ring), warps 2,3: none, warps 4..: tile pairs
    ARK_HD static constexpr int pair_of_warp(int w) { return w == 0 ? 0 : (w == 1 ? NW - 1 : (w < 4 ? -1 : w - 3)); }
};

template <bool VISC, int TX, int NW>
struct ArkMarch3 {
    double *UR, *PBb, *PBa, *FB, *TB, *YB, *GB, *EB;
    const double* Ucol[2];               // host emulation only: the two own columns of the input state
    const void* tmap;                    // tensor map of the input state (TMA tile loads of the UR ring)
    int tx, ty;                          // box origin in the padded array (columns, rows)
    unsigned long long* mbar;            // the block's three mbarriers (one per UR slot)
    unsigned phase;                      // parity bit of each slot's next completion
    double* Ocur;                        // row a, plane q-1 of the output state (row b: + px)
    long long pstride, fs;
    int px;
    int s, ca;                           // exchange slot (pair * RX + lane); UR column of row a (row b: + RX)
    int k0, k1;
    bool inU[2], want_rate;
    int xwrap;                           // periodic x: offset of the ghost copy of this column (+nx, -nx) or 0
    bool xwrap_any;                      // warp-uniform: some lane of the warp owns a column with a ghost copy
    int uq, un, unn, pc, pn;             // ring slots of planes q, q+1, q+2 (UR); q, q+1 (PB)
    // z pipelines of the two columns: the acoustic z face (q-1|q) stays in registers, everything else is parked in
    // TMEM between its uses (primitives of planes q-1 / q / q+1 in two alternating slots, U~(q-1), the running
    // update of plane q-1, the centred differences of plane q-1)
    ArkFace zlo[2];
    unsigned tm;                         // TMEM address of this thread's scratch columns
    int tcur;                            // TMEM primitive slot of plane q (the other one holds q-1, then q+1)
    ark_u64 rate_max;
    // general path only (GEN; see ark_step.cuh): array-valued potential, read straight from global memory
    const double* php;                   // plane q+1 of the padded potential at this lane's column (row 0 of the array)
    int pho[4];                          // row offsets (doubles) of rows a-1, a, b, b+1, clamped to the padded array
    double phc[2];                       // Phi(q) of the own two columns
    double ghz[2];                       // -(Phi(q) - Phi(q-1)) of the own two columns: the z face (q-1|q)
    double ghyu_prev;                    // -(Phi_{b+1} - Phi_b) at plane q-1: the high-y face of row b, used one plane later
};

template <bool VISC, int TX, int NW>
ARK_DEV void ark_ring_issue3(const ArkMarch3<VISC, TX, NW>& M, int k, int slot) {
    using C = ArkCfg3<VISC, TX, NW>;
#ifndef ARK_HOST_EMU
    if (threadIdx.x == 0) {
        unsigned long long* bar = M.mbar + slot;
        ark_mbar_expect_tx(bar, 5u * C::NCOL * (unsigned)sizeof(double));
        ark_tma_load_4d(M.UR + slot * 5 * C::NCOL, M.tmap, M.tx, M.ty, k + ARK_NG, 0, bar);
    }
#else
    for (int r = 0; r < 2; ++r) {
        const double* c = M.Ucol[r] + M.pstride * (long long)k;
        double* d = M.UR + slot * 5 * C::NCOL + M.ca + r * C::RX;
        for (int f = 0; f < 5; ++f) d[f * C::NCOL] = c[f * M.fs];
    }
#endif
}

template <bool VISC, int TX, int NW>
ARK_DEV void ark_ring_wait3(ArkMarch3<VISC, TX, NW>& M, int slot) {
#ifndef ARK_HOST_EMU
    ark_mbar_wait(M.mbar + slot, (M.phase >> slot) & 1u);
    M.phase ^= 1u << slot;
#else
    (void)M; (void)slot;
#endif
}

// Block barrier (B) of a plane: a plain __syncthreads at the point where a warp's faces / differences / primitives are in
// shared memory; work that only needs the warp's own data (the parked z pipeline, five of the six dissipative face fluxes)
// is ordered BEFORE it.  Measured and rejected (profiles/r02_step_kernel.md): a split arrive / wait on an mbarrier
// (5.367 vs 5.356 ms at 512^3) and unrolling the steady plane loop twice (5.60 vs 5.14 ms: the unrolled tile loop, 37 KB,
// no longer fits the 32 KB instruction cache).
#ifndef ARK_RING_EARLY
#define ARK_RING_EARLY 1
#endif
template <bool VISC, int TX, int NW>
ARK_DEV void ark_bar_arrive(ArkMarch3<VISC, TX, NW>& M) {
    (void)M;
    __syncthreads();
}
template <bool VISC, int TX, int NW>
ARK_DEV void ark_bar_wait(ArkMarch3<VISC, TX, NW>& M) { (void)M; }   // (the point where a neighbour's data is first read)

template <bool VISC, int TX, int NW>
ARK_DEV ArkPrim ark_march_prims3(const ArkParams& P, const ArkMarch3<VISC, TX, NW>& M, int col, int slot) {
    constexpr int NCOL = ArkCfg3<VISC, TX, NW>::NCOL;
    const double* u = M.UR + slot * 5 * NCOL + col;
    return ark_prim_fast(P, u[0], u[NCOL], u[2 * NCOL], u[3 * NCOL], u[4 * NCOL]);
}

// TMEM scratch layout of one thread (32-bit columns; a double = 2 columns): primitives [slot][row][8] stored as
// (u,v,w,T,rho,p,rc,irc) so that the q-1 plane's u,v,w,T come back with one 4-double load; U~ [row][8 (5 used)];
// running update [row][8 (5 used)]; differences dxw,dxu,dyw,dyv [row][4].  144 columns per thread.
#define ARK_TM_PR(slot, r) (16u * (unsigned)(2 * (slot) + (r)))
#define ARK_TM_TP(r) (64u + 16u * (unsigned)(r))
#define ARK_TM_AC(r) (96u + 16u * (unsigned)(r))
#define ARK_TM_GZ(r) (128u + 8u * (unsigned)(r))
#define ARK_TM_COLS 144
ARK_DEV void ark_tm_put_prim(unsigned a, const ArkPrim& w) { ark_tm_st8(a, w.u, w.v, w.w, w.T, w.rho, w.p, w.rc, w.irc); }
ARK_DEV void ark_tm_get_prim(unsigned a, ArkPrim& w) { ark_tm_ld8(a, w.u, w.v, w.w, w.T, w.rho, w.p, w.rc, w.irc); }
ARK_DEV void ark_tm_put5(unsigned a, const double* v) { ark_tm_st4(a, v[0], v[1], v[2], v[3]); ark_tm_st1(a + 8, v[4]); }
ARK_DEV void ark_tm_get5(unsigned a, double* v) { ark_tm_ld4(a, v[0], v[1], v[2], v[3]); ark_tm_ld1(a + 8, v[4]); }

// Full flux through a face with normal along axis DN (1: x, 2: y, 3: z): upwind transport of U~ on u* plus the
// acoustic part (0, Pi* e_d, Pi* u*) minus the dissipative flux.
// vis = (tau_dn, tau_da, tau_db, energy flux) in the face's own (normal, a, b) order, see ark_visc_face.
template <int DN, bool VISC>
ARK_DEV void ark_face_flux(double* F, bool left, const double* TL, const double* TR, double us, double pi, const ArkVisc& vis) {
    const double t0 = left ? TL[0] : TR[0], t1 = left ? TL[1] : TR[1], t2 = left ? TL[2] : TR[2], t3 = left ? TL[3] : TR[3],
                 t4 = left ? TL[4] : TR[4];
    F[0] = t0 * us;
    F[1] = DN == 1 ? t1 * us + pi : t1 * us;
    F[2] = DN == 2 ? t2 * us + pi : t2 * us;
    F[3] = DN == 3 ? t3 * us + pi : t3 * us;
    F[4] = (t4 + pi) * us;
    if (VISC) {
        // component order of vis: normal, a, b with (a,b) = (y,z) for x, (x,z) for y, (x,y) for z
        if (DN == 1) { F[1] -= vis.t0; F[2] -= vis.t1; F[3] -= vis.t2; }
        if (DN == 2) { F[1] -= vis.t1; F[2] -= vis.t0; F[3] -= vis.t2; }
        if (DN == 3) { F[1] -= vis.t1; F[2] -= vis.t2; F[3] -= vis.t0; }
        F[4] -= vis.fe;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Lock-step helpers: N independent instances of the same formula, written statement by statement over all
// instances, so that the instruction stream alternates between independent dependency chains (a thread owns two
// rows: the fp64 pipe has a ~9-cycle dependent-issue latency and a warp scheduler holds only 2-3 of these warps).
// The arithmetic of each instance is exactly that of ark_prim_fast / ark_face / ark_visc_face / ark_face_flux.
// ------------------------------------------------------------------------------------------------------------
template <int N>
ARK_DEV void ark_rcp_n(const double* x, double* r) {
#ifndef ARK_IEEE_RCP
    double y[N], e[N];
#pragma unroll
    for (int i = 0; i < N; ++i) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y[i]) : "d"(x[i]));
#pragma unroll
    for (int i = 0; i < N; ++i) e[i] = fma(-x[i], y[i], 1.0);
#pragma unroll
    for (int i = 0; i < N; ++i) e[i] = fma(e[i], e[i], e[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = fma(y[i], e[i], y[i]);
#else
    for (int i = 0; i < N; ++i) r[i] = 1.0 / x[i];
#endif
}

template <int N>
ARK_DEV void ark_rsqrt_n(const double* x, double* r) {
#ifndef ARK_IEEE_RCP
    double y[N], e[N], t[N];
#pragma unroll
    for (int i = 0; i < N; ++i) asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y[i]) : "d"(x[i]));
#pragma unroll
    for (int i = 0; i < N; ++i) t[i] = -x[i] * y[i];
#pragma unroll
    for (int i = 0; i < N; ++i) e[i] = fma(t[i], y[i], 1.0);
#pragma unroll
    for (int i = 0; i < N; ++i) t[i] = fma(0.375, e[i], 0.5);
#pragma unroll
    for (int i = 0; i < N; ++i) e[i] = y[i] * e[i];
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = fma(e[i], t[i], y[i]);
#else
    for (int i = 0; i < N; ++i) r[i] = 1.0 / sqrt(x[i]);
#endif
}

// primitives of N cells from their conserved values U[i] = (rho, mx, my, mz, E)
template <int N>
ARK_DEV void ark_prim_fast_n(const ArkParams& P, const double (*U)[5], ArkPrim* q) {
    double hm2[N], ggr[N], rho[N], rinv[N], ei[N], gpr[N];
#pragma unroll
    for (int i = 0; i < N; ++i) rho[i] = U[i][0];
#pragma unroll
    for (int i = 0; i < N; ++i) hm2[i] = 0.5 * (U[i][1] * U[i][1] + U[i][2] * U[i][2] + U[i][3] * U[i][3]);
#pragma unroll
    for (int i = 0; i < N; ++i) ggr[i] = (P.gamma * P.gm1) * rho[i];
    ark_rcp_n<N>(rho, rinv);
#pragma unroll
    for (int i = 0; i < N; ++i) { q[i].rho = rho[i]; q[i].u = U[i][1] * rinv[i]; q[i].v = U[i][2] * rinv[i]; q[i].w = U[i][3] * rinv[i]; }
#pragma unroll
    for (int i = 0; i < N; ++i) ei[i] = U[i][4] - hm2[i] * rinv[i];
#pragma unroll
    for (int i = 0; i < N; ++i) { q[i].p = P.gm1 * ei[i]; gpr[i] = ggr[i] * ei[i]; }
    double irc[N];
    ark_rsqrt_n<N>(gpr, irc);
#pragma unroll
    for (int i = 0; i < N; ++i) { q[i].irc = irc[i]; q[i].rc = gpr[i] * irc[i]; q[i].T = q[i].p * rinv[i]; }
}

struct ArkFaceIn { double gh, rhoL, unL, pL, rcL, ircL, rhoR, unR, pR, rcR, ircR; };
ARK_DEV ArkFaceIn ark_face_in(double gh, double rhoL, double unL, double pL, double rcL, double ircL,
                              double rhoR, double unR, double pR, double rcR, double ircR) {
    ArkFaceIn f = {gh, rhoL, unL, pL, rcL, ircL, rhoR, unR, pR, rcR, ircR};
    return f;
}

template <int N>
ARK_DEV void ark_face_n(int theta_on, const ArkFaceIn* in, ArkFace* f) {
    bool lg[N];
    double a[N], i2a[N], dp[N], um[N], du[N], pm[N], ath[N];
#pragma unroll
    for (int i = 0; i < N; ++i) lg[i] = in[i].rcL > in[i].rcR;
#pragma unroll
    for (int i = 0; i < N; ++i) { a[i] = ARK_K_IMPEDANCE * (lg[i] ? in[i].rcL : in[i].rcR); i2a[i] = (0.5 / ARK_K_IMPEDANCE) * (lg[i] ? in[i].ircL : in[i].ircR); }
#pragma unroll
    for (int i = 0; i < N; ++i) { f[i].S = (0.5 * in[i].gh) * (in[i].rhoL + in[i].rhoR); dp[i] = in[i].pR - in[i].pL; um[i] = in[i].unL + in[i].unR; }
#pragma unroll
    for (int i = 0; i < N; ++i) { dp[i] = dp[i] - f[i].S; du[i] = in[i].unR - in[i].unL; pm[i] = in[i].pL + in[i].pR; }
#pragma unroll
    for (int i = 0; i < N; ++i) f[i].us = 0.5 * um[i] - dp[i] * i2a[i];
#pragma unroll
    for (int i = 0; i < N; ++i) ath[i] = a[i];
    if (theta_on) {
        double icL[N], icR[N], ma[N];
#pragma unroll
        for (int i = 0; i < N; ++i) { icL[i] = in[i].rhoL * in[i].ircL; icR[i] = in[i].rhoR * in[i].ircR; }
#pragma unroll
        for (int i = 0; i < N; ++i) ma[i] = fabs(f[i].us) * (icL[i] < icR[i] ? icL[i] : icR[i]);
#pragma unroll
        for (int i = 0; i < N; ++i) ath[i] = a[i] * (ma[i] < 1.0 ? ma[i] : 1.0);
    }
#pragma unroll
    for (int i = 0; i < N; ++i) f[i].pi = 0.5 * pm[i] - 0.5 * ath[i] * du[i];
}

struct ArkViscIn { double dn_n, dn_a, dn_b, tra_n, tra_a, trb_n, trb_b, ub_n, ub_a, ub_b, dT; };
template <int N>
ARK_DEV void ark_visc_face_n(const ArkViscCoef& K, const ArkViscIn* in, ArkVisc* r) {
#pragma unroll
    for (int i = 0; i < N; ++i) { r[i].t0 = K.c43 * in[i].dn_n - K.c23t * (in[i].tra_a + in[i].trb_b); r[i].t1 = K.cn * in[i].dn_a + K.ct * in[i].tra_n; r[i].t2 = K.cn * in[i].dn_b + K.ct * in[i].trb_n; }
#pragma unroll
    for (int i = 0; i < N; ++i) r[i].fe = 0.5 * (r[i].t0 * in[i].ub_n + r[i].t1 * in[i].ub_a + r[i].t2 * in[i].ub_b) + K.kh * in[i].dT;
}

// N-wide flux through faces with normal along axis DN (see ark_face_flux)
template <int DN, bool VISC, int N>
ARK_DEV void ark_face_flux_n(double (*F)[5], const bool* left, const double* const* TL, const double* const* TR, const double* us,
                             const double* pi, const ArkVisc* vis) {
    double t[N][5];
#pragma unroll
    for (int f = 0; f < 5; ++f)
#pragma unroll
        for (int i = 0; i < N; ++i) t[i][f] = left[i] ? TL[i][f] : TR[i][f];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        F[i][0] = t[i][0] * us[i];
        F[i][1] = DN == 1 ? t[i][1] * us[i] + pi[i] : t[i][1] * us[i];
        F[i][2] = DN == 2 ? t[i][2] * us[i] + pi[i] : t[i][2] * us[i];
        F[i][3] = DN == 3 ? t[i][3] * us[i] + pi[i] : t[i][3] * us[i];
    }
#pragma unroll
    for (int i = 0; i < N; ++i) F[i][4] = (t[i][4] + pi[i]) * us[i];
    if (VISC) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            if (DN == 1) { F[i][1] -= vis[i].t0; F[i][2] -= vis[i].t1; F[i][3] -= vis[i].t2; }
            if (DN == 2) { F[i][1] -= vis[i].t1; F[i][2] -= vis[i].t0; F[i][3] -= vis[i].t2; }
            if (DN == 3) { F[i][1] -= vis[i].t1; F[i][2] -= vis[i].t2; F[i][3] -= vis[i].t0; }
            F[i][4] -= vis[i].fe;
        }
    }
}

// Ring warps, one plane EARLY.  A ring warp (one row, no lock-step partner, sharing its scheduler with two tile warps) is
// the last to reach barrier B if it computes all its faces there; but the x-, (a|b) and low-y faces and the x differences
// of plane p only need primitives of plane p, which exist one iteration before they are used.  So they are computed
// between barriers B and C of the previous iteration, where the ring warp has little else to do and would wait for the
// tile warps, and parked in its unused TMEM columns; before barrier B only the z face (which needs plane p+1) is left.
// Same functions, same inputs: the results are bit-identical.  w: primitives of the ring row at plane p; pslot: PB / EB
// slot of plane p.
#define ARK_TM_EARLY 64u                                       // 11 doubles in the (unused) U~ columns of a ring warp
template <bool VISC, bool GXY, int TX, int NW, int ROLE>
ARK_DEV void ark_ring_early3(const ArkParams& P, ArkMarch3<VISC, TX, NW>& M, const ArkPrim& w, int pslot) {
    using C = ArkCfg3<VISC, TX, NW>;
    constexpr int RX = C::RX, NP = C::NP, NT = C::NS;
    constexpr int NFE = ROLE == 0 ? 2 : 3;
    const int s = M.s;
    const double ghx = GXY ? P.D.gh[0] : 0.0, ghy = GXY ? P.D.gh[1] : 0.0;
    const double* e = M.EB + (pslot * 2 + (ROLE == 0 ? 0 : 1)) * 5 * RX + (s % RX);     // the edge row next to the ring row
    const double lr = ark_xl(w.rho), Lu = ark_xl(w.u), lp = ark_xl(w.p), lrc = ark_xl(w.rc), lirc = ark_xl(w.irc);
    ArkFaceIn in[NFE];
    ArkFace out[NFE];
    in[0] = ark_face_in(ghx, lr, Lu, lp, lrc, lirc, w.rho, w.u, w.p, w.rc, w.irc);
    if (ROLE == 0) in[1] = ark_face_in(ghy, e[0], e[RX], e[2 * RX], e[3 * RX], e[4 * RX], w.rho, w.v, w.p, w.rc, w.irc);   // (edge | ring)
    else           in[1] = ark_face_in(ghy, w.rho, w.v, w.p, w.rc, w.irc, e[0], e[RX], e[2 * RX], e[3 * RX], e[4 * RX]);   // (ring | edge)
    if (ROLE == 2) {
        const double* n = M.PBb + pslot * NP * NT + (s - RX);                           // row a-1 (pair below)
        in[NFE - 1] = ark_face_in(ghy, n[0], n[2 * NT], n[4 * NT], n[5 * NT], n[6 * NT], w.rho, w.v, w.p, w.rc, w.irc);
    }
    ark_face_n<NFE>(P.theta, in, out);
    double dxu = 0.0, dxv = 0.0;
    if (VISC) { dxu = ark_xr(w.u) - Lu; dxv = ark_xr(w.v) - ark_xl(w.v); }
    const unsigned a = M.tm + ARK_TM_EARLY;
    ark_tm_st4(a, out[0].us, out[0].pi, out[0].S, out[1].us);
    ark_tm_st4(a + 8, out[1].pi, out[1].S, dxu, dxv);
    if (ROLE == 2) { ark_tm_st2(a + 16, out[2].us, out[2].pi); ark_tm_st1(a + 20, out[2].S); }
}

// GXY: gravity may have x / y components (false: only g_z, the x and y source terms vanish at compile time)
// PAR >= 0: the parity of the plane inside the two-fold unrolled steady loop, which makes the alternating slots (TMEM
// primitive slot, PB slot) compile-time constants; -1: read them from M
template <bool VISC, bool GXY, bool GEN, int TX, int NW, int ROLE, bool STEADY, int PAR = -1>
ARK_DEV void ark_plane3(const ArkParams& P, const ArkStepConst& K, ArkMarch3<VISC, TX, NW>& M, const int q) {
    static_assert(!GEN || GXY, "the general path keeps all gravity components");
    using C = ArkCfg3<VISC, TX, NW>;
    constexpr int RX = C::RX, NCOL = C::NCOL, NP = C::NP, NT = C::NS;   // NT: stride of the exchange arrays
    constexpr int R0 = ROLE == 0 ? 1 : 0, R1 = ROLE == 2 ? 0 : 1, NA = R1 - R0 + 1;   // active (ring / tile) rows of the pair
    const int s = M.s;
    const double lam = K.lam;
    const bool do_update = STEADY || (q >= M.k0 && q < M.k1);     // plane q is an output plane of this chunk
    const bool has_zlo = STEADY || q >= M.k0;                     // face (q-1|q) bounds an output plane
    const bool completes = STEADY || q > M.k0;                    // plane q-1 is completed and stored here
    const bool gx = GXY && P.D.g_on[0], gy = GXY && P.D.g_on[1];
    const double ghx = GXY ? P.D.gh[0] : 0.0, ghy = GXY ? P.D.gh[1] : 0.0;
    const unsigned tm = M.tm;
    constexpr bool EARLY = ARK_RING_EARLY && ROLE != 1 && !GEN;   // ring warps: see ark_ring_early3
    const int tcur = PAR >= 0 ? PAR : M.tcur;
    const int pc = PAR >= 0 ? PAR : M.pc, pn = pc ^ 1;
    // GEN: every face has its own -(Phi_R - Phi_L) in place of g_d h; the gravity work
    // is lam * that difference * the inflowing mass flux, or, for Appendix B (P.eform == 1), replaced by lam (uS)_i
    const bool PH = GEN && P.phi != nullptr;
    const bool eformB = GEN && P.eform == 1;
    const bool wk = !eformB;
    double ghxl[2] = {ghx, ghx}, ghxh[2] = {ghx, ghx}, ghzh[2] = {P.D.gh[2], P.D.gh[2]}, ghyi = ghy, ghyl = ghy, ghyu = ghy;
    if (PH) {
        const double* pq1 = M.php;                        // plane q+1
        const double* pq0 = M.php - M.pstride;            // plane q
        ghyi = M.phc[0] - M.phc[1];
        if (ROLE != 0) ghyl = pq0[M.pho[0]] - M.phc[0];
        if (ROLE != 2) ghyu = M.phc[1] - pq0[M.pho[3]];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const double phn = pq1[M.pho[1 + r]];
            ghzh[r] = M.phc[r] - phn;
            ghxl[r] = ark_xl(M.phc[r]) - M.phc[r];
            ghxh[r] = ark_xr(ghxl[r]);
            M.phc[r] = phn;                               // (the differences of plane q are complete: rotate)
        }
    }

    // ---------------- S1: primitives of plane q (parked in TMEM one iteration ago) and, for the viscous z stencil,
    // u,v,w,T of plane q-1; prefetch plane q+2; primitives of plane q+1 of the own two columns
    ArkPrim wc[2], wn[2];
    double wm[2][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}};
    ark_tm_wait_st();
#pragma unroll
    for (int r = R0; r <= R1; ++r) ark_tm_get_prim(tm + ARK_TM_PR(tcur, r), wc[r]);
    double er[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};           // ring warps: what ark_ring_early3 parked for this plane
    if (EARLY) {
        ark_tm_ld4(tm + ARK_TM_EARLY, er[0], er[1], er[2], er[3]);
        ark_tm_ld4(tm + ARK_TM_EARLY + 8, er[4], er[5], er[6], er[7]);
        if (ROLE == 2) { ark_tm_ld2(tm + ARK_TM_EARLY + 16, er[8], er[9]); ark_tm_ld1(tm + ARK_TM_EARLY + 20, er[10]); }
    }
    if (VISC) {
#pragma unroll
        for (int r = R0; r <= R1; ++r) ark_tm_ld4(tm + ARK_TM_PR(tcur ^ 1, r), wm[r][0], wm[r][1], wm[r][2], wm[r][3]);
    }
    if (STEADY || q + 2 <= M.k1 + 1) ark_ring_issue3(M, q + 2, M.unn);
    ark_ring_wait3(M, M.un);
    {
        // (ring pairs: only the ring row; the primitives of their edge row come from the edge warps through EB)
        double U[2][5];
        const double* u = M.UR + M.un * 5 * NCOL + M.ca;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
#pragma unroll
            for (int r = R0; r <= R1; ++r) U[r][f] = u[f * NCOL + r * RX];
        }
        ark_prim_fast_n<NA>(P, U + R0, wn + R0);
    }
    if (ROLE != 2) {                                              // row b: all primitives, for the pair above
        double* p = M.PBb + pn * NP * NT + s;
        p[0] = wn[1].rho; p[NT] = wn[1].u; p[2 * NT] = wn[1].v; p[3 * NT] = wn[1].w;
        p[4 * NT] = wn[1].p; p[5 * NT] = wn[1].rc; p[6 * NT] = wn[1].irc;
        if (VISC) p[7 * NT] = wn[1].T;
    }
    if (VISC && ROLE != 0) {                                      // row a: velocity, for the centred differences of the pair below
        double* p = M.PBa + pn * 3 * NT + s;
        p[0] = wn[0].u; p[NT] = wn[0].v; p[2 * NT] = wn[0].w;
    }
    ark_tm_wait_ld();
    // (no barrier: S2 reads the neighbours' primitives of plane q, written one iteration ago)

    // ---------------- S2: acoustic faces of plane q, centred velocity differences
    ArkFace fx[2], zhi[2], fyl = {0, 0, 0}, fyi;
    double Lu[2] = {0, 0}, Lv[2] = {0, 0}, Lw[2] = {0, 0}, LT[2] = {0, 0};
    double dxu[2] = {0, 0}, dxv[2] = {0, 0}, dxw[2] = {0, 0}, dyu[2] = {0, 0}, dyv[2] = {0, 0}, dyw[2] = {0, 0};
    double dzu[2] = {0, 0}, dzv[2] = {0, 0}, dzw[2] = {0, 0};
    ArkPrim Bm;                                                   // row a-1 (pair below)
    Bm.rho = Bm.u = Bm.v = Bm.w = Bm.p = Bm.rc = Bm.irc = Bm.T = 0;
    if (ROLE != 0) {
        const double* n = M.PBb + pc * NP * NT + (s - RX);
        Bm.rho = n[0]; Bm.u = n[NT]; Bm.v = n[2 * NT]; Bm.w = n[3 * NT]; Bm.p = n[4 * NT]; Bm.rc = n[5 * NT]; Bm.irc = n[6 * NT];
        if (VISC) Bm.T = n[7 * NT];
    }
    if (ROLE != 1 && !EARLY) {
        // the edge row of a ring pair (row a of pair 0, row b of pair NW-1) only enters the (a|b) face
        constexpr int RE = ROLE == 0 ? 0 : 1;
        const double* e = M.EB + (pc * 2 + RE) * 5 * RX + (s % RX);
        wc[RE].rho = e[0]; wc[RE].v = e[RX]; wc[RE].p = e[2 * RX]; wc[RE].rc = e[3 * RX]; wc[RE].irc = e[4 * RX];
    }
    if (EARLY) {
        // x-, (a|b), low-y faces and x differences of this plane come from TMEM (computed one iteration ago); only the
        // z face is computed here
        constexpr int r = R0;
        const ArkPrim& c = wc[r];
        const ArkFaceIn zin = ark_face_in(P.D.gh[2], c.rho, c.w, c.p, c.rc, c.irc, wn[r].rho, wn[r].w, wn[r].p, wn[r].rc, wn[r].irc);
        ark_face_n<1>(P.theta, &zin, &zhi[r]);
        fx[r].us = er[0]; fx[r].pi = er[1]; fx[r].S = er[2];
        fyi.us = er[3]; fyi.pi = er[4]; fyi.S = er[5];
        if (ROLE == 2) { fyl.us = er[8]; fyl.pi = er[9]; fyl.S = er[10]; }
    } else {
        // faces in lock-step: x- and z+ of the active rows, low-y of row a (not for the low ring pair), (a|b)
        constexpr int NF = 2 * NA + (ROLE != 0 ? 2 : 1);
        ArkFaceIn in[NF];
        ArkFace out[NF];
        double lr[2], lp[2], lrc[2], lirc[2];
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            lr[r] = ark_xl(wc[r].rho); Lu[r] = ark_xl(wc[r].u); lp[r] = ark_xl(wc[r].p); lrc[r] = ark_xl(wc[r].rc); lirc[r] = ark_xl(wc[r].irc);
        }
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            const ArkPrim& c = wc[r];
            in[r - R0] = ark_face_in(GEN ? ghxl[r] : ghx, lr[r], Lu[r], lp[r], lrc[r], lirc[r], c.rho, c.u, c.p, c.rc, c.irc);
            in[NA + r - R0] = ark_face_in(GEN ? ghzh[r] : P.D.gh[2], c.rho, c.w, c.p, c.rc, c.irc, wn[r].rho, wn[r].w, wn[r].p, wn[r].rc, wn[r].irc);
        }
        {
            const ArkPrim &a = wc[0], &b = wc[1];
            in[2 * NA] = ark_face_in(GEN ? ghyi : ghy, a.rho, a.v, a.p, a.rc, a.irc, b.rho, b.v, b.p, b.rc, b.irc);
            if (ROLE != 0) in[NF - 1] = ark_face_in(GEN ? ghyl : ghy, Bm.rho, Bm.v, Bm.p, Bm.rc, Bm.irc, a.rho, a.v, a.p, a.rc, a.irc);
        }
        ark_face_n<NF>(P.theta, in, out);
#pragma unroll
        for (int r = R0; r <= R1; ++r) { fx[r] = out[r - R0]; zhi[r] = out[NA + r - R0]; }
        fyi = out[2 * NA];
        if (ROLE != 0) fyl = out[NF - 1];
    }
    if (ROLE != 0) {                                              // low-y face of row a -> the pair below (its high-y face)
        M.FB[s] = fyl.us; M.FB[NT + s] = fyl.pi;
        if (gy) M.FB[2 * NT + s] = fyl.S;
    }
    if (VISC) {
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            const ArkPrim& c = wc[r];
            if (EARLY) { dxu[r] = er[6]; dxv[r] = er[7]; }
            else {
                Lv[r] = ark_xl(c.v);
                dxu[r] = ark_xr(c.u) - Lu[r];
                dxv[r] = ark_xr(c.v) - Lv[r];
            }
            dzv[r] = wn[r].v - wm[r][1];
            dzw[r] = wn[r].w - wm[r][2];
            if (ROLE == 1) {
                Lw[r] = ark_xl(c.w);
                LT[r] = ark_xl(c.T);
                dxw[r] = ark_xr(c.w) - Lw[r];
                dzu[r] = wn[r].u - wm[r][0];
            }
        }
    }
    // plane q+1 is parked for the next iteration (its slot held plane q-1, which is in registers now)
#pragma unroll
    for (int r = R0; r <= R1; ++r) ark_tm_put_prim(tm + ARK_TM_PR(tcur ^ 1, r), wn[r]);
    if (VISC && ROLE == 1) {                                      // centred y differences of the two tile rows
        const double* n = M.PBa + pc * 3 * NT + (s + RX);        // row b+1 (pair above)
        dyu[0] = wc[1].u - Bm.u; dyv[0] = wc[1].v - Bm.v; dyw[0] = wc[1].w - Bm.w;
        dyu[1] = n[0] - wc[0].u; dyv[1] = n[NT] - wc[0].v; dyw[1] = n[2 * NT] - wc[0].w;
    }
    if (VISC && ROLE != 2) {                                      // row b's differences feed the low-y face of the pair above
        M.GB[s] = dxv[1]; M.GB[NT + s] = dxu[1]; M.GB[2 * NT + s] = dzv[1]; M.GB[3 * NT + s] = dzw[1];
    }
    ark_bar_arrive(M);                                            // (B) faces, differences (and prims q+1) written

    // ---------------- between arrive and wait: what needs no neighbour -- the parked z pipeline of the tile rows and the
    // dissipative fluxes (reading A6) through the x-, z- and (a|b) faces, in lock-step
    double Tp[2][5], acc[2][5], gpz[2][4];
    ArkVisc vyl = {0, 0, 0, 0}, vx[2] = {{0, 0, 0, 0}, {0, 0, 0, 0}}, vz[2] = {{0, 0, 0, 0}, {0, 0, 0, 0}}, vyi = {0, 0, 0, 0};
    if (ROLE == 1) {
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            if (VISC) ark_tm_ld4(tm + ARK_TM_GZ(r), gpz[r][0], gpz[r][1], gpz[r][2], gpz[r][3]);
            ark_tm_get5(tm + ARK_TM_TP(r), Tp[r]);
            ark_tm_get5(tm + ARK_TM_AC(r), acc[r]);
        }
        ark_tm_wait_ld();
        if (VISC) {
            ArkViscIn in[5];
            ArkVisc out[5];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const ArkPrim& c = wc[r];
                // face (i-1 | i), normal x, transverse a = y, b = z
                const ArkViscIn v1 = {c.u - Lu[r], c.v - Lv[r], c.w - Lw[r], ark_xl(dyu[r]) + dyu[r], ark_xl(dyv[r]) + dyv[r],
                                      ark_xl(dzu[r]) + dzu[r], ark_xl(dzw[r]) + dzw[r], Lu[r] + c.u, Lv[r] + c.v, Lw[r] + c.w, c.T - LT[r]};
                in[r] = v1;
                // face (q-1 | q), normal z, transverse a = x, b = y
                const double um = wm[r][0], vm = wm[r][1], wmm = wm[r][2], Tm = wm[r][3];
                const ArkViscIn v2 = {c.w - wmm, c.u - um, c.v - vm, gpz[r][0] + dxw[r], gpz[r][1] + dxu[r], gpz[r][2] + dyw[r],
                                      gpz[r][3] + dyv[r], wmm + c.w, um + c.u, vm + c.v, c.T - Tm};
                in[2 + r] = v2;
            }
            const ArkPrim &a = wc[0], &b = wc[1];                 // face (a | b), normal y, transverse a = x, b = z
            const ArkViscIn v3 = {b.v - a.v, b.u - a.u, b.w - a.w, dxv[0] + dxv[1], dxu[0] + dxu[1], dzv[0] + dzv[1],
                                  dzw[0] + dzw[1], a.v + b.v, a.u + b.u, a.w + b.w, b.T - a.T};
            in[4] = v3;
            ark_visc_face_n<5>(P.D.KV, in, out);
            vx[0] = out[0]; vx[1] = out[1]; vz[0] = out[2]; vz[1] = out[3]; vyi = out[4];
        }
    }
    ark_bar_wait(M);                                              // (B) the neighbours' faces, differences visible

    // ---------------- S3: acoustic update U~(q), PAPER.md:158-160 (+ reading A3 for the energy)
    ArkFace fyu = {0, 0, 0};                                      // high-y face of row b = low-y face of the pair above
    if (ROLE != 2) {
        fyu.us = M.FB[s + RX]; fyu.pi = M.FB[NT + s + RX];
        if (gy) fyu.S = M.FB[2 * NT + s + RX];
    }
    double Uc[2][5], Ut[2][5], Six[2] = {0, 0}, Siy[2] = {0, 0}, Siz[2] = {0, 0};
    double usxh[2], pixh[2], Sxh[2] = {0, 0}, suS[2] = {0, 0};
#pragma unroll
    for (int r = 0; r < 2; ++r) { for (int f = 0; f < 5; ++f) Uc[r][f] = Ut[r][f] = 0.0; usxh[r] = pixh[r] = 0.0; }
    {
        // lock-step over the active rows
        double sdu[2], sdpu[2], den[2], iLt[2];
        const ArkFace* yl[2] = {&fyl, &fyi};                      // low-y / high-y acoustic face of rows a, b
        const ArkFace* yh[2] = {&fyi, &fyu};
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            const double* uc = M.UR + M.uq * 5 * NCOL + M.ca + r * RX;
            Uc[r][0] = wc[r].rho; Uc[r][1] = uc[NCOL]; Uc[r][2] = uc[2 * NCOL]; Uc[r][3] = uc[3 * NCOL]; Uc[r][4] = uc[4 * NCOL];
            usxh[r] = ark_xr(fx[r].us); pixh[r] = ark_xr(fx[r].pi);
            if (gx) { Sxh[r] = ark_xr(fx[r].S); Six[r] = 0.5 * (fx[r].S + Sxh[r]); }   // S_i = (S_low + S_high)/2
        }
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            if (gy) Siy[r] = 0.5 * (yl[r]->S + yh[r]->S);
            Siz[r] = 0.5 * (zhi[r].S + M.zlo[r].S);
            sdu[r] = (usxh[r] - fx[r].us) + (yh[r]->us - yl[r]->us) + (zhi[r].us - M.zlo[r].us);
        }
#pragma unroll
        for (int r = R0; r <= R1; ++r) den[r] = 1.0 + lam * sdu[r];
        ark_rcp_n<NA>(den + R0, iLt + R0);
#pragma unroll
        for (int r = R0; r <= R1; ++r)
            sdpu[r] = (pixh[r] * usxh[r] - fx[r].pi * fx[r].us) + (yh[r]->pi * yh[r]->us - yl[r]->pi * yl[r]->us)
                    + (zhi[r].pi * zhi[r].us - M.zlo[r].pi * M.zlo[r].us);
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            Ut[r][1] = GXY ? (Uc[r][1] - lam * (pixh[r] - fx[r].pi) + lam * Six[r]) : (Uc[r][1] - lam * (pixh[r] - fx[r].pi));
            Ut[r][2] = GXY ? (Uc[r][2] - lam * (yh[r]->pi - yl[r]->pi) + lam * Siy[r]) : (Uc[r][2] - lam * (yh[r]->pi - yl[r]->pi));
            Ut[r][3] = (Uc[r][3] - lam * (zhi[r].pi - M.zlo[r].pi) + lam * Siz[r]);
            if (eformB) {
                // Appendix B (reading A24): (uS)_i = 1/2 (u* S at the high face + u* S at the low face), per axis
                suS[r] = 0.5 * (usxh[r] * Sxh[r] + fx[r].us * fx[r].S) + 0.5 * (yh[r]->us * yh[r]->S + yl[r]->us * yl[r]->S)
                       + 0.5 * (zhi[r].us * zhi[r].S + M.zlo[r].us * M.zlo[r].S);
                Ut[r][4] = ((Uc[r][4] + lam * suS[r]) - lam * sdpu[r]);
            } else {
                Ut[r][4] = (Uc[r][4] - lam * sdpu[r]);
            }
        }
#pragma unroll
        for (int r = R0; r <= R1; ++r) {
            Ut[r][0] = Uc[r][0] * iLt[r]; Ut[r][1] *= iLt[r]; Ut[r][2] *= iLt[r]; Ut[r][3] *= iLt[r]; Ut[r][4] *= iLt[r];
        }
    }
    if (ROLE != 2) {                                              // U~ of row b: upwind state of the pair above's low-y face
        double* tb = M.TB + s;
        tb[0] = Ut[1][0]; tb[NT] = Ut[1][1]; tb[2 * NT] = Ut[1][2]; tb[3 * NT] = Ut[1][3]; tb[4 * NT] = Ut[1][4];
    }

    // dissipative flux through the low-y face of row a (needs the differences of the pair below)
    if (VISC && ROLE != 0) {
        const double* g = M.GB + (s - RX);                       // dxv,dxu,dzv,dzw of row a-1
        const ArkPrim& c = wc[0];
        const ArkViscIn v = {c.v - Bm.v, c.u - Bm.u, c.w - Bm.w, g[0] + dxv[0], g[NT] + dxu[0], g[2 * NT] + dzv[0],
                             g[3 * NT] + dzw[0], Bm.v + c.v, Bm.u + c.u, Bm.w + c.w, c.T - Bm.T};
        ark_visc_face_n<1>(P.D.KV, &v, &vyl);
    }

    if (ROLE == 1) {
        // ---- z face (q-1|q): completes plane q-1
        double Gz[2][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
        if (has_zlo) {
            double fyh[5] = {0, 0, 0, 0, 0};                      // flux through the high-y face of row b at plane q-1
            if (completes) { const double* y = M.YB + (s + RX); fyh[0] = y[0]; fyh[1] = y[NT]; fyh[2] = y[2 * NT]; fyh[3] = y[3 * NT]; fyh[4] = y[4 * NT]; }
            {
                // upwind on u* (reading A10): U~(q-1) or U~(q) of the own column
                const bool left[2] = {ark_nonneg(M.zlo[0].us), ark_nonneg(M.zlo[1].us)};
                const double* TL[2] = {Tp[0], Tp[1]};
                const double* TR[2] = {Ut[0], Ut[1]};
                const double us[2] = {M.zlo[0].us, M.zlo[1].us}, pi[2] = {M.zlo[0].pi, M.zlo[1].pi};
                ark_face_flux_n<3, VISC, 2>(Gz, left, TL, TR, us, pi, vz);
            }
            if (completes) {
                // U^{n+1}(q-1) = running update - lam * (high-z flux) [- lam * (high-y flux) for row b] + gravity work
                double out[2][5];
#pragma unroll
                for (int f = 0; f < 5; ++f) { out[0][f] = acc[0][f] - lam * Gz[0][f]; out[1][f] = acc[1][f] - lam * Gz[1][f]; }
#pragma unroll
                for (int f = 0; f < 5; ++f) out[1][f] -= lam * fyh[f];
                if (GEN) {
                    if (wk && gy) out[1][4] += lam * M.ghyu_prev * ark_neg_part(fyh[0]);
                    if (wk && P.D.g_on[2]) { out[0][4] += lam * M.ghz[0] * ark_neg_part(Gz[0][0]); out[1][4] += lam * M.ghz[1] * ark_neg_part(Gz[1][0]); }
                } else {
                    if (gy) out[1][4] += K.dt * P.g[1] * ark_neg_part(fyh[0]);
                    if (P.D.g_on[2]) { out[0][4] += K.dt * P.g[2] * ark_neg_part(Gz[0][0]); out[1][4] += K.dt * P.g[2] * ark_neg_part(Gz[1][0]); }
                }
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    if (M.inU[r]) {
                        double* __restrict__ o = M.Ocur + r * M.px;          // plane q-1 of this column
                        o[0] = out[r][0]; o[M.fs] = out[r][1]; o[2 * M.fs] = out[r][2]; o[3 * M.fs] = out[r][3]; o[4 * M.fs] = out[r][4];
                    }
                    if (M.xwrap_any && M.inU[r] && M.xwrap != 0) {
                        // periodic x: the first / last two columns also fill the opposite ghost columns of the new
                        // state, so that the next step needs no x ghost-fill launch
                        double* __restrict__ o = M.Ocur + r * M.px + M.xwrap;
                        o[0] = out[r][0]; o[M.fs] = out[r][1]; o[2 * M.fs] = out[r][2]; o[3 * M.fs] = out[r][3]; o[4 * M.fs] = out[r][4];
                    }
                }
                if (M.want_rate) {
                    // CFL rate of the new state (reading A4), both rows in lock-step
                    double rinv[2], s1[2], ke[2], c2[2], ic[2], rho2[2] = {out[0][0], out[1][0]};
                    ark_rcp_n<2>(rho2, rinv);
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        s1[r] = (fabs(out[r][1]) + fabs(out[r][2]) + fabs(out[r][3])) * rinv[r];
                        ke[r] = 0.5 * (out[r][1] * out[r][1] + out[r][2] * out[r][2] + out[r][3] * out[r][3]) * rinv[r];
                    }
#pragma unroll
                    for (int r = 0; r < 2; ++r) c2[r] = P.gamma * (P.gm1 * (out[r][4] - ke[r])) * rinv[r];
                    ark_rsqrt_n<2>(c2, ic);
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        const double rate = (s1[r] + 3.0 * (c2[r] * ic[r])) * P.D.inv_h + P.D.dcoef * rinv[r];
                        const ark_u64 rr = ark_rate_bits(rate) & 0x7fffffffffffffffULL;
                        M.rate_max = ark_umax(M.rate_max, M.inU[r] ? rr : 0ULL);
                    }
                }
            }
        }
        // U~(q) and the differences of plane q replace those of plane q-1 in TMEM
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            ark_tm_put5(tm + ARK_TM_TP(r), Ut[r]);
            if (VISC) ark_tm_st4(tm + ARK_TM_GZ(r), dxw[r], dxu[r], dyw[r], dyv[r]);
        }
        // ---- x faces and the (a|b) face of plane q: start the running update of plane q
        if (do_update) {
            double TL[2][5], Fl[2][5], Fh[2][5];
#pragma unroll
            for (int f = 0; f < 5; ++f) { TL[0][f] = ark_xl(Ut[0][f]); TL[1][f] = ark_xl(Ut[1][f]); }
            {
                const bool left[2] = {ark_nonneg(fx[0].us), ark_nonneg(fx[1].us)};
                const double* tl[2] = {TL[0], TL[1]};
                const double* tr[2] = {Ut[0], Ut[1]};
                const double us[2] = {fx[0].us, fx[1].us}, pi[2] = {fx[0].pi, fx[1].pi};
                ark_face_flux_n<1, VISC, 2>(Fl, left, tl, tr, us, pi, vx);
            }
#pragma unroll
            for (int f = 0; f < 5; ++f) { Fh[0][f] = ark_xr(Fl[0][f]); Fh[1][f] = ark_xr(Fl[1][f]); }
            double F[1][5];
            {
                const bool left[1] = {ark_nonneg(fyi.us)};
                const double* tl[1] = {Ut[0]};
                const double* tr[1] = {Ut[1]};
                ark_face_flux_n<2, VISC, 1>(F, left, tl, tr, &fyi.us, &fyi.pi, &vyi);
            }
            // low z face enters with +lam*G_z and the gravity work dt g_z max(m,0); sources lam*S_i
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                acc[r][0] = (Uc[r][0] - lam * (Fh[r][0] - Fl[r][0])) + lam * Gz[r][0];
                acc[r][1] = GXY ? (Uc[r][1] - lam * (Fh[r][1] - Fl[r][1]) + lam * Six[r]) + lam * Gz[r][1] : (Uc[r][1] - lam * (Fh[r][1] - Fl[r][1])) + lam * Gz[r][1];
                acc[r][2] = GXY ? (Uc[r][2] - lam * (Fh[r][2] - Fl[r][2]) + lam * Siy[r]) + lam * Gz[r][2] : (Uc[r][2] - lam * (Fh[r][2] - Fl[r][2])) + lam * Gz[r][2];
                acc[r][3] = (Uc[r][3] - lam * (Fh[r][3] - Fl[r][3])) + lam * Gz[r][3];
                if (GEN) {
                    double work = 0.0;                                  // (in units of lam)
                    if (eformB) work = suS[r];
                    else if (gx) work = ghxl[r] * ark_pos_part(Fl[r][0]) + ghxh[r] * ark_neg_part(Fh[r][0]);
                    acc[r][4] = (Uc[r][4] - lam * (Fh[r][4] - Fl[r][4]) + lam * work) + lam * Gz[r][4];
                } else if (GXY) {
                    double work = 0.0;
                    if (gx) work = P.g[0] * (ark_pos_part(Fl[r][0]) + ark_neg_part(Fh[r][0]));
                    acc[r][4] = (Uc[r][4] - lam * (Fh[r][4] - Fl[r][4]) + K.dt * work) + lam * Gz[r][4];
                } else {
                    acc[r][4] = (Uc[r][4] - lam * (Fh[r][4] - Fl[r][4])) + lam * Gz[r][4];
                }
                if (P.D.g_on[2]) {
                    acc[r][3] += lam * Siz[r];
                    if (GEN) { if (wk) acc[r][4] += lam * M.ghz[r] * ark_pos_part(Gz[r][0]); }
                    else acc[r][4] += K.dt * P.g[2] * ark_pos_part(Gz[r][0]);
                }
            }
#pragma unroll
            for (int f = 0; f < 5; ++f) { acc[0][f] -= lam * F[0][f]; acc[1][f] += lam * F[0][f]; }
            if (gy && wk) {
                const double cy = GEN ? lam * ghyi : K.dt * P.g[1];
                acc[0][4] += cy * ark_neg_part(F[0][0]);
                acc[1][4] += cy * ark_pos_part(F[0][0]);
            }
            ark_tm_put5(tm + ARK_TM_AC(1), acc[1]);               // row b is complete but for its high-y / high-z faces
        }
    }
    // ring warps: the faces of plane q+1 that need no plane q+2, while the tile warps are busy with plane q
    if (EARLY) ark_ring_early3<VISC, GXY, TX, NW, ROLE>(P, M, wn[R0], pn);
    __syncthreads();                                              // (C) U~(q) of the pair below visible

    // ---------------- S4: low-y face of row a
    if (ROLE != 0 && do_update) {
        const double* tb = M.TB + (s - RX);
        double TL[5], F[5];
        TL[0] = tb[0]; TL[1] = tb[NT]; TL[2] = tb[2 * NT]; TL[3] = tb[3 * NT]; TL[4] = tb[4 * NT];
        ark_face_flux<2, VISC>(F, ark_nonneg(fyl.us), TL, Ut[0], fyl.us, fyl.pi, vyl);
        double* y = M.YB + s;
        y[0] = F[0]; y[NT] = F[1]; y[2 * NT] = F[2]; y[3 * NT] = F[3]; y[4 * NT] = F[4];
        if (ROLE == 1) {
#pragma unroll
            for (int f = 0; f < 5; ++f) acc[0][f] += lam * F[f];
            if (gy && wk) acc[0][4] += (GEN ? lam * ghyl : K.dt * P.g[1]) * ark_pos_part(F[0]);
            ark_tm_put5(tm + ARK_TM_AC(0), acc[0]);
        }
    }

    // rotate the pipelines; the output pointer follows plane q
    if (ROLE == 1) {
        M.Ocur += M.pstride;
#ifndef ARK_HOST_EMU
        asm volatile("" : "+l"(M.Ocur));
#endif
    }
#pragma unroll
    for (int r = R0; r <= R1; ++r) M.zlo[r] = zhi[r];
    if (GEN) { M.ghz[0] = ghzh[0]; M.ghz[1] = ghzh[1]; M.ghyu_prev = ghyu; M.php += M.pstride; }
    { const int t3 = M.uq; M.uq = M.un; M.un = M.unn; M.unn = t3; }
    if (PAR < 0) {
        M.tcur ^= 1;
        const int t2 = M.pc; M.pc = M.pn; M.pn = t2;
    }
}

template <bool VISC, bool GXY, bool GEN, int TX, int NW, int ROLE>
ARK_DEV void ark_march3(const ArkParams& P, const ArkStepConst& K, ArkMarch3<VISC, TX, NW>& M) {
    int q = M.k0 - 1;
    for (; q <= M.k0; ++q) ark_plane3<VISC, GXY, GEN, TX, NW, ROLE, false>(P, K, M, q);   // k0-1, k0
    for (; q < M.k1; ++q) ark_plane3<VISC, GXY, GEN, TX, NW, ROLE, true>(P, K, M, q);     // k0+1 .. k1-1
    for (; q <= M.k1; ++q) ark_plane3<VISC, GXY, GEN, TX, NW, ROLE, false>(P, K, M, q);   // k1
}

// prologue (planes k0-2, k0-1; k0 in flight) and plane loop of one row pair
template <bool VISC, bool GXY, bool GEN, int TX, int NW, int ROLE>
ARK_DEV void ark_run_pair3(const ArkParams& P, const ArkStepConst& K, ArkMarch3<VISC, TX, NW>& M) {
    using C = ArkCfg3<VISC, TX, NW>;
    constexpr int RX = C::RX, NS = C::NS;
    ark_ring_wait3(M, 0);
    ark_ring_wait3(M, 1);
    ArkPrim wc0[2];
    constexpr int R0 = ROLE == 0 ? 1 : 0, R1 = ROLE == 2 ? 0 : 1;   // active (ring / tile) rows of the pair
#pragma unroll
    for (int r = R0; r <= R1; ++r) {
        const ArkPrim wm = ark_march_prims3(P, M, M.ca + r * RX, 0);
        wc0[r] = ark_march_prims3(P, M, M.ca + r * RX, 1);
        ark_tm_put_prim(M.tm + ARK_TM_PR(1, r), wm);              // plane k0-2 (the "q-1" slot of the first iteration)
        ark_tm_put_prim(M.tm + ARK_TM_PR(0, r), wc0[r]);          // plane k0-1
        double ghz0 = P.D.gh[2];
        if (GEN) {
            if (P.phi) {                                  // M.php points at plane k0: planes k0-2, k0-1 of this column
                const double phm = M.php[M.pho[1 + r] - 2 * M.pstride];
                M.phc[r] = M.php[M.pho[1 + r] - M.pstride];
                ghz0 = phm - M.phc[r];
            }
            M.ghz[r] = ghz0;
        }
        M.zlo[r] = ark_face(P.theta, ghz0, wm.rho, wm.w, wm.p, wm.rc, wm.irc, wc0[r].rho, wc0[r].w, wc0[r].p, wc0[r].rc, wc0[r].irc);
        if (ROLE == 1) {
            const double zero5[5] = {0, 0, 0, 0, 0};
            ark_tm_put5(M.tm + ARK_TM_TP(r), zero5);
            ark_tm_put5(M.tm + ARK_TM_AC(r), zero5);
            ark_tm_st4(M.tm + ARK_TM_GZ(r), 0.0, 0.0, 0.0, 0.0);
        }
    }
    if (ROLE != 2) {
        double* p = M.PBb + M.pc * C::NP * NS + M.s;
        const ArkPrim& w = wc0[1];
        p[0] = w.rho; p[NS] = w.u; p[2 * NS] = w.v; p[3 * NS] = w.w; p[4 * NS] = w.p; p[5 * NS] = w.rc; p[6 * NS] = w.irc;
        if (VISC) p[7 * NS] = w.T;
    }
    if (VISC && ROLE != 0) {
        double* p = M.PBa + M.pc * 3 * NS + M.s;
        p[0] = wc0[0].u; p[NS] = wc0[0].v; p[2 * NS] = wc0[0].w;
    }
    __syncthreads();                                  // primitives of plane k0-1 visible to the neighbours
    if (ARK_RING_EARLY && ROLE != 1 && !GEN) ark_ring_early3<VISC, GXY, TX, NW, ROLE>(P, M, wc0[ROLE == 0 ? 1 : 0], M.pc);   // plane k0-1
    ark_march3<VISC, GXY, GEN, TX, NW, ROLE>(P, K, M);
    ark_tm_wait_st();
}

// Edge rows 0 and RY-1 of the region only provide primitives for one acoustic face each (the (a|b) face of the ring
// pair next to them).  Warps 2 and 3 of warpgroup 0 compute them, one plane ahead like every other row, and hand
// rho, v, p, rho c, 1/(rho c) to the ring warps through EB: the ring warps, which run alone on their schedulers next to
// two tile warps and are on the critical path of every block barrier, carry one row instead of two.
template <bool VISC, int TX, int NW>
ARK_DEV void ark_edge_prims3(const ArkParams& P, const ArkMarch3<VISC, TX, NW>& M, int e, int uslot, int pslot) {
    using C = ArkCfg3<VISC, TX, NW>;
    const ArkPrim w = ark_march_prims3(P, M, M.ca + e * C::RX, uslot);
    double* d = M.EB + (pslot * 2 + e) * 5 * C::RX + (M.s % C::RX);
    d[0] = w.rho; d[C::RX] = w.v; d[2 * C::RX] = w.p; d[3 * C::RX] = w.rc; d[4 * C::RX] = w.irc;
}

template <bool VISC, int TX, int NW>
ARK_DEV void ark_run_edge3(const ArkParams& P, ArkMarch3<VISC, TX, NW>& M, int e) {
    ark_ring_wait3(M, 0);
    ark_ring_wait3(M, 1);
    ark_edge_prims3(P, M, e, 1, M.pc);                // plane k0-1
    __syncthreads();
    for (int q = M.k0 - 1; q <= M.k1; ++q) {
        if (q + 2 <= M.k1 + 1) ark_ring_issue3(M, q + 2, M.unn);   // (a no-op on the GPU: thread 0 issues the TMA loads)
        ark_ring_wait3(M, M.un);
        ark_edge_prims3(P, M, e, M.un, M.pn);         // plane q+1
        { const int t3 = M.uq; M.uq = M.un; M.un = M.unn; M.unn = t3; }
        { const int t2 = M.pc; M.pc = M.pn; M.pn = t2; }
        ark_bar_arrive(M);
        ark_bar_wait(M);
        __syncthreads();
    }
}

#ifndef ARK_HOST_EMU
template <int N> ARK_DEV void ark_setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> ARK_DEV void ark_setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
#else
template <int N> ARK_DEV void ark_setmaxnreg_dec() {}
template <int N> ARK_DEV void ark_setmaxnreg_inc() {}
#endif

template <bool VISC, bool GXY, bool GEN, int TX, int NW>
ARK_DEV void ark_step3d_pairs(const ArkParams& P, const double* __restrict__ Uin, double* __restrict__ Uout, double dt_value,
                              const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk, double* smem,
                              const void* tmap) {
    using C = ArkCfg3<VISC, TX, NW>;
    constexpr int RX = C::RX, TY = C::TY;
    ArkMarch3<VISC, TX, NW> M;
    M.UR = smem + C::UR_OFF;
    M.PBb = smem + C::PBB_OFF;
    M.PBa = smem + C::PBA_OFF;
    M.FB = smem + C::FB_OFF;
    M.TB = smem + C::TB_OFF;
    M.YB = smem + C::YB_OFF;
    M.GB = smem + C::GB_OFF;
    M.EB = smem + C::EB_OFF;
    ark_u64* red = (ark_u64*)(smem + C::RED_OFF);
    M.mbar = (unsigned long long*)(smem + C::MBAR_OFF);

    const int t = threadIdx.x;
    const int lane = t % RX, warp = t / RX, pair = C::pair_of_warp(warp);
    const int prow = pair >= 0 ? pair : (warp == 2 ? 0 : NW - 1);   // warps 2, 3: the edge row of the low / high ring pair
    M.s = prow * RX + lane;
    M.ca = (2 * prow) * RX + lane;
    const int gi = blockIdx.x * TX - 2 + lane, gja = blockIdx.y * TY - 2 + 2 * prow;   // interior-based cell coordinates (row a)
    if (zchunk > 0) {                                           // uniform chunks (tests); 0: the table of ark_create
        M.k0 = blockIdx.z * zchunk;
        M.k1 = M.k0 + zchunk < P.nz ? M.k0 + zchunk : P.nz;
    } else {
        M.k0 = P.zb[blockIdx.z];
        M.k1 = P.zb[blockIdx.z + 1];
    }
    const bool tile = pair >= 1 && pair <= NW - 2;
    const bool inx = lane >= 2 && lane < 2 + TX && gi < P.nx;
    M.inU[0] = tile && inx && gja < P.ny;
    M.inU[1] = tile && inx && gja + 1 < P.ny;
    M.want_rate = rate_scratch != nullptr;
    M.xwrap = 0;
    if (P.bc[0][0] == ARK_BCK_PERIODIC && lane >= 2 && lane < 2 + TX) {
        if (gi < 2) M.xwrap = P.nx;
        else if (gi >= P.nx - 2 && gi < P.nx) M.xwrap = -P.nx;
    }
#ifndef ARK_HOST_EMU
    M.xwrap_any = __any_sync(0xffffffffu, M.xwrap != 0);
#else
    M.xwrap_any = true;
#endif

    const ArkStepConst K = ark_step_const(P, dt_value, dt_dev);
    M.pstride = (long long)P.px * P.py;
    M.fs = P.fstride;
    M.px = P.px;
    {
        // host emulation reads its own columns; columns beyond the padded array (ragged tiles) load a valid cell
        const int li = gi < P.nx + 2 ? gi : P.nx + 1;
        for (int r = 0; r < 2; ++r) {
            const int gj = gja + r, lj = gj < P.ny + 2 ? gj : P.ny + 1;
            M.Ucol[r] = Uin + (long long)(li + ARK_XOFF) + (long long)P.px * (long long)(lj + ARK_NG) + M.pstride * (long long)P.offz;
        }
        const int lo = gi < P.nx ? gi : P.nx - 1, ljo = gja < P.ny ? gja : P.ny - 1;
        M.Ocur = Uout + (long long)(lo + ARK_XOFF) + (long long)P.px * (long long)(ljo + ARK_NG) + M.pstride * (long long)(P.offz + M.k0 - 2);
    }
    M.php = nullptr;
    M.phc[0] = M.phc[1] = M.ghz[0] = M.ghz[1] = M.ghyu_prev = 0.0;
    M.pho[0] = M.pho[1] = M.pho[2] = M.pho[3] = 0;
    if (GEN && P.phi) {
        const int li = gi < P.nx + 2 ? gi : P.nx + 1;
        for (int i = 0; i < 4; ++i) {
            int gj = gja - 1 + i;
            gj = gj < -ARK_NG ? -ARK_NG : (gj < P.ny + 2 ? gj : P.ny + 1);
            M.pho[i] = P.px * (gj + ARK_NG);
        }
        M.php = P.phi + (li + ARK_XOFF) + M.pstride * (long long)(P.offz + M.k0);   // plane q+1 at q = k0-1
    }
    M.tmap = tmap;
    M.tx = (int)(blockIdx.x * TX) - 2 + ARK_XOFF;
    M.ty = (int)(blockIdx.y * TY) - 2 + ARK_NG;
    M.phase = 0;
    unsigned tmem_base = 0;
#ifndef ARK_HOST_EMU
    unsigned* tm_slot = (unsigned*)(smem + C::MBAR_OFF + 3);
    if (t == 0) {
        for (int s3 = 0; s3 < 3; ++s3) ark_mbar_init(M.mbar + s3, 1);
        ark_mbar_fence_init();
    }
    if (t < 32) ark_tm_alloc_all(tm_slot);            // the whole TMEM of the SM (one block per SM)
    ark_tm_fence_before_sync();
    __syncthreads();
    ark_tm_fence_after_sync();
    tmem_base = *tm_slot;
    // TMEM scratch of this thread: lane quarter of the warp, column range of the warp within the quarter
    // (warp-uniform by construction; the OR-reduction hands it to the compiler as a uniform-register value, so that
    // every tcgen05.ld / st addresses tmem[UR + imm] without a per-instruction register -> uniform-register move)
    M.tm = __reduce_or_sync(0xffffffffu, tmem_base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)((warp >> 2) * ARK_TM_COLS));
#else
    M.tm = 0; (void)tmem_base;
#endif
    M.tcur = 0;
    M.rate_max = 0;

    // ring slots at q = k0-1: UR planes (k0-2,) k0-1, k0, k0+1 -> slots (0,) 1, 2, 0
    M.uq = 1; M.un = 2; M.unn = 0;
    M.pc = 0; M.pn = 1;
    for (int s3 = 0; s3 < 3; ++s3) ark_ring_issue3(M, M.k0 - 2 + s3, s3);

    if (warp < 4) {
        ark_setmaxnreg_dec<C::REG_RING>();
        if (pair == 0)           ark_run_pair3<VISC, GXY, GEN, TX, NW, 0>(P, K, M);
        else if (pair == NW - 1) ark_run_pair3<VISC, GXY, GEN, TX, NW, 2>(P, K, M);
        else                     ark_run_edge3<VISC, TX, NW>(P, M, warp == 2 ? 0 : 1);   // warps 2, 3: the edge rows
    } else {
        ark_setmaxnreg_inc<C::REG_TILE>();
        ark_run_pair3<VISC, GXY, GEN, TX, NW, 1>(P, K, M);
    }

    if (rate_scratch) {
        // block-wide max of the rate bit patterns -> one double per block
        ark_u64 m = M.rate_max;
#ifndef ARK_HOST_EMU
        for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        const int wl = t & 31, wid = t >> 5;
        if (wl == 0) red[wid] = m;
        __syncthreads();
        if (wid == 0) {
            m = wl < C::NWARP ? red[wl] : 0;
            for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        }
#else
        m = ark_emu_block_umax(m);
        (void)red;
#endif
        if (t == 0) rate_scratch[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = ark_rate_from_bits(m);
    }
#ifndef ARK_HOST_EMU
    ark_tm_fence_before_sync();
    __syncthreads();
    if (t < 32) ark_tm_free_all(tmem_base);
#endif
}

template <bool VISC, bool GXY, bool GEN, int TX, int NW>
ARK_GLOBAL void
#ifndef ARK_HOST_EMU
__launch_bounds__(ArkCfg3<VISC, TX, NW>::NT, 1)
#endif
ark_k_step3(const ArkParams P, const double* __restrict__ Uin, double* __restrict__ Uout, double dt_value,
            const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk ARK_TMAP_PARAM) {
#ifndef ARK_HOST_EMU
    extern __shared__ __align__(128) unsigned char ark_smem_raw[];
    double* smem = reinterpret_cast<double*>(ark_smem_raw);
#else
    ARK_DYN_SMEM(smem);
#endif
    ark_step3d_pairs<VISC, GXY, GEN, TX, NW>(P, Uin, Uout, dt_value, dt_dev, rate_scratch, zchunk, smem, ARK_TMAP_ARG);
}
