// ark_step.cuh -- the fused full-step kernel (acoustic + transport + dissipative + update + CFL epilogue).
//
// One launch advances U^n -> U^{n+1}: every conserved field is read once and written once
// (80 B per cell update in 3D, 64 B in 2D); all face quantities, velocity gradients and the intermediate
// state U~ live in registers / shared memory only.
//
// Decomposition ("2.5-D marching"): a block owns a TX x TY tile of (x,y) columns plus a 2-cell halo
// (region RX x RY = (TX+4) x (TY+4)) and marches along z over a chunk of planes.  The product build uses
// TX = 28, so RX = 32: ONE WARP PER REGION ROW 1..RY-2 (the two edge rows 0 and RY-1 only need primitives and are
// the second column of the ring-row threads).  Every role in the kernel depends on the ROW only (ring row / tile row),
// i.e. is warp-uniform and a compile-time parameter of the plane loop: no lane is predicated off inside a phase (the
// 4 halo lanes of a row compute values nobody consumes); only the final stores and the CFL rate carry a per-lane
// predicate.
//
// What persists from plane to plane --
//   UR  U^n of planes q, q+1, q+2 in shared memory, filled two planes ahead by ONE TMA tensor tile load per block
//       and plane (cp.async.bulk.tensor, 4-D box RX x RY x 1 x 5 fields, completion on an mbarrier): the HBM
//       prefetch costs no registers, no LSU wavefronts and one instruction of one thread
//   PB  primitives of planes q, q+1 in shared memory (the x/y neighbours read them)
//   TB  U~ of planes q-1, q in shared memory
//   registers: the own column's primitives of plane q and u,v,w,T of plane q-1, the running update acc[5], the low
//   z face and four velocity differences.
//
// Per plane q one iteration does (2 block barriers):
//   S1  primitives of plane q+1 (own column, from the UR ring)          -> PB
//   S2  acoustic faces x-, y- of plane q (neighbours from PB), z face (q|q+1) from the own column   -> FB
//       cell-centred velocity differences of plane q                                               -> GB
//   --- barrier B
//   S3  acoustic update U~(q) on tile + 1 ring       -> TB
//       viscous / heat fluxes through the x-, y- faces of plane q      -> VB ; z- face in registers
//   --- barrier C
//   S4  transport fluxes (upwind on u*) of the in-plane faces of plane q and of the
//       z face (q-1|q); completes and stores U^{n+1}(q-1); folds the CFL rate of the new state into a
//       per-block maximum (integer max on the bit patterns, NaN-propagating).
// What only the x neighbour consumes (high-x acoustic face, the left cell's differences, the high-x viscous flux) is
// exchanged by warp shuffle and never touches shared memory.
#pragma once
#include "ark_device.cuh"

#define ARK_NPRIM 8   // rho,u,v,w,p,rc,irc,T

template <int NDIM, bool VISC, int TX, int TY>
struct ArkStepCfg {
    static constexpr int RX = TX + 4, RY = TY + 4, NCOL = RX * RY;
    // 3D: one thread per column of rows 1..RY-2; the two edge rows 0 and RY-1 (primitives only) are the second
    // column of the threads of the ring rows 1 and RY-2, whose own work is light.  2D: one thread per column.
    static constexpr int NTHR = NDIM == 3 ? RX * (RY - 2) : NCOL;
    static constexpr int NT = ((NTHR + 31) / 32) * 32;
    static constexpr int NP = VISC ? 8 : 7;                          // T only feeds the heat flux
    static constexpr int PSLOTS = NDIM == 3 ? 2 : 1;                 // primitives of planes q, q+1
    static constexpr int UR = NDIM == 3 ? 15 : 0;                    // [3][5]
    static constexpr int FBN = NDIM == 3 ? 4 : 6;                    // 3D recomputes the gravity face terms S
    static constexpr int TSLOTS = NDIM == 3 ? 2 : 1;
    // shared memory (doubles per column): UR, PB[PSLOTS][NP], FB, TB[TSLOTS][5], GB[7], VB[8] (+ 32 for the reduction)
    static constexpr int PER_COL = UR + PSLOTS * NP + FBN + TSLOTS * 5 + (VISC ? 15 : 0);
    static constexpr int SMEM_DOUBLES = PER_COL * NCOL + 32 + 3 * RY;   // + reduction + per row: 3 mbarriers (UR slots), phase counter
    static constexpr size_t SMEM_BYTES = (size_t)SMEM_DOUBLES * sizeof(double);
};

// sign tests on the integer pipe (the fp64 pipe is the bottleneck of this kernel): for u* >= 0 the paper's
// upwind choice is the left cell (reading A10); -0.0 picks the right cell, whose flux is
// multiplied by that same zero.
#ifndef ARK_HOST_EMU
ARK_DEV bool ark_nonneg(double x) { return __double2hiint(x) >= 0; }
#else
ARK_DEV bool ark_nonneg(double x) { return (int)(__double_as_longlong(x) >> 32) >= 0; }
#endif
ARK_DEV double ark_pos_part(double x) { return ark_nonneg(x) ? x : 0.0; }   // max(x, 0)
ARK_DEV double ark_neg_part(double x) { return ark_nonneg(x) ? 0.0 : x; }   // min(x, 0)

struct ArkVisc { double t0, t1, t2, fe; };

// Exchange with the x neighbours by warp shuffle when a region row is exactly one warp (RX == 32): what only the
// left / right neighbour consumes (high-x acoustic face, the left cell's centred differences, the high-x viscous
// flux) then never touches shared memory.  Other tile widths and the host emulation use the shared arrays.
#ifndef ARK_HOST_EMU
#define ARK_XSHFL(RX) ((RX) == 32)
ARK_DEV double ark_from_left(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
ARK_DEV double ark_from_right(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
#else
#define ARK_XSHFL(RX) false
ARK_DEV double ark_from_left(double v) { return v; }
ARK_DEV double ark_from_right(double v) { return v; }
#endif

// Dissipative flux through a face with unit normal along axis d (tau = mu(grad u + grad u^T)
// + eta div u I, eta = -2/3 mu; divergence form, Fourier flux; stencil = reading A6).
//   dn_*  : (u_d, u_a, u_b)_R - (..)_L                        normal differences (un-normalised)
//   tra_n, tra_a : sum over the two adjacent cells of the centred difference along transverse axis a of
//                  u_d and u_a   -> d_a u_d and d_a u_a at the face are tr/(4h)
//   trb_n, trb_b : same along transverse axis b for u_d and u_b
//   ub_*  : (u_d, u_a, u_b)_L + (..)_R                        (2 x face velocity)
//   dT    : T_R - T_L
// tau_dd = 2 mu d_d u_d - 2/3 mu div u = (4/3)(mu/h) dn_n - (2/3)(mu/4h)(tra_a + trb_b)
// tau_da = mu (d_d u_a + d_a u_d)      = (mu/h) dn_a + (mu/4h) tra_n
// Returns tau_{d,.} ordered (normal, a, b) and the energy flux tau.ubar + kappa dT/h.
ARK_DEV ArkVisc ark_visc_face(const ArkViscCoef& K, double dn_n, double dn_a, double dn_b,
                              double tra_n, double tra_a, double trb_n, double trb_b,
                              double ub_n, double ub_a, double ub_b, double dT) {
    ArkVisc r;
    r.t0 = K.c43 * dn_n - K.c23t * (tra_a + trb_b);
    r.t1 = K.cn * dn_a + K.ct * tra_n;
    r.t2 = K.cn * dn_b + K.ct * trb_n;
    r.fe = 0.5 * (r.t0 * ub_n + r.t1 * ub_a + r.t2 * ub_b) + K.kh * dT;
    return r;
}

// CFL rate of one cell of the NEW state for the fused epilogue (reading A4), as the bit pattern of |rate|
// (see ark_rate_bits): one fast reciprocal and one fast rsqrt per cell.
ARK_DEV ark_u64 ark_rate_epilogue(const ArkParams& P, int ndim, double rho, double mx, double my, double mz, double E,
                                  double inv_h, double dcoef) {
    const double rinv = ark_rcp(rho);
    const double s = (fabs(mx) + fabs(my) + fabs(mz)) * rinv;
    const double ke = 0.5 * (mx * mx + my * my + mz * mz) * rinv;
    const double c2 = P.gamma * (P.gm1 * (E - ke)) * rinv;
    const double c = c2 * ark_rsqrt(c2);
    const double r = (s + (double)ndim * c) * inv_h + dcoef * rinv;
    return ark_rate_bits(r) & 0x7fffffffffffffffULL;
}

// per-thread constants of a step: only the time step itself (it may come from device memory, ark_run); everything
// else that is uniform sits in P.D (constant bank)
struct ArkStepConst { double dt, lam; };

ARK_DEV ArkStepConst ark_step_const(const ArkParams& P, double dt_value, const double* __restrict__ dt_dev) {
    ArkStepConst c;
    c.dt = dt_dev ? dt_dev[1] : dt_value;
    c.lam = c.dt / P.h;
    return c;
}

// Transport through the two faces of one in-plane axis of the cell in column tc (stride sd between neighbours):
// F = U~_up u* + (0, Pi* e_d, Pi* u*); adds F_{d+} - F_{d-} to dG and the gravity
// work g_d (min(m_{d+},0) + max(m_{d-},0)) to work (reading A13).  T points at U~ of plane q,
// component stride cs.  DN = index of the normal momentum (1: x, 2: y).
template <int NDIM, int DN>
ARK_DEV void ark_transport_axis(const double* __restrict__ T, int cs, int tc, int sd, double usl, double pil, double ush,
                                double pih, bool g_on, double g, double* dG, double& work, bool first) {
    const int nl = ark_nonneg(usl) ? tc - sd : tc, nh = ark_nonneg(ush) ? tc : tc + sd;
    const double ml = T[nl] * usl, mh = T[nh] * ush;
    // each face flux is formed first (normal momentum: U~_up u* + Pi*), then differenced: the order of the flux
    // form (11), which keeps the O(1) pressure terms bit-compatible with a plain evaluation (reading A20)
    double d[5];
    d[0] = mh - ml;
    d[1] = DN == 1 ? (T[cs + nh] * ush + pih) - (T[cs + nl] * usl + pil) : T[cs + nh] * ush - T[cs + nl] * usl;
    d[2] = DN == 2 ? (T[2 * cs + nh] * ush + pih) - (T[2 * cs + nl] * usl + pil) : T[2 * cs + nh] * ush - T[2 * cs + nl] * usl;
    d[3] = NDIM == 3 ? T[3 * cs + nh] * ush - T[3 * cs + nl] * usl : 0.0;
    d[4] = (T[4 * cs + nh] + pih) * ush - (T[4 * cs + nl] + pil) * usl;
    if (first) { for (int f = 0; f < 5; ++f) dG[f] = d[f]; }
    else       { for (int f = 0; f < 5; ++f) dG[f] += d[f]; }
    if (g_on) work += g * (ark_pos_part(ml) + ark_neg_part(mh));
}

// ------------------------------------------------------------------------------------------------------------
// 3D body.  The march is specialised by ROW ROLE (a compile-time parameter of the whole plane loop, chosen once
// per thread and warp-uniform when RX == 32) so that no role test, no predicate and no dummy initialisation is
// left inside an iteration:
//   ROLE 1  ring rows 1, RY-2 : primitives, acoustic faces, centred differences, U~, viscous low-y face; each thread
//                               also keeps the primitives of the EDGE row next to it (row 0 / RY-1: prefetch,
//                               primitives and, for row RY-1, its low-y face) -- the edge rows have no threads
//   ROLE 2  tile rows 2..RY-3 : + viscous x / z faces, transport, update, store, CFL rate
// and by STEADY (planes k0+1 .. k1-1, where every chunk-boundary condition is known) vs. the generic first and
// last iterations.  Every role executes the same two barriers per plane.
// ------------------------------------------------------------------------------------------------------------
template <bool VISC, int TX, int TY>
struct ArkMarch {
    double *UR, *PB, *FB, *TB, *GB, *VB;
    const double* Ucol;
    const double* Ucol2;                 // ring rows: the edge column (row 0 or RY-1) this thread also serves
    const void* tmap;                    // tensor map of the input state (TMA tile loads of the UR ring)
    int tx, ty;                          // box origin in the padded array (columns, rows)
    unsigned long long* mbar;            // the block's three mbarriers (one per UR slot)
    unsigned phase;                      // parity bit of each slot's next completion
    double* Ocur;                        // tile rows: plane q-1 of the own column in the output state
    long long pstride, fs;
    int tc, tc2, k0, k1;
    bool inU, want_rate, top;            // top: ring row RY-2 (its edge row RY-1 owns a low-y face)
    int uq, un, unn, pc, pn, tq;         // ring slots of planes q, q+1, q+2 (UR); q, q+1 (PB); q (TB)
    ArkPrim wc;                          // primitives of the own column at plane q
    double wm[4];                        // u,v,w,T of the own column at plane q-1 (viscous z stencil)
    ArkFace zlo;                         // acoustic z face (q-1|q)
    double acc[5];                       // U^{n+1}(q-1) minus its high-z flux
    double gpz[4];                       // dxw,dxu,dyw,dyv of the own column at q-1 (viscous z face)
    ark_u64 rate_max;
};

// U^n(k) of the whole region -> UR[slot].  GPU: thread 0 of the block issues one TMA tile load (box RX x RY x 1 plane
// x 5 fields, laid out in shared memory exactly as UR[slot][field][row][column]) completing on the block's mbarrier
// of that slot.  Host emulation: every thread copies its own column(s) synchronously.
template <bool VISC, int TX, int TY>
ARK_DEV void ark_ring_issue(const ArkMarch<VISC, TX, TY>& M, int k, int slot, bool edge) {
    using C = ArkStepCfg<3, VISC, TX, TY>;
    constexpr int NCOL = C::NCOL;
#ifndef ARK_HOST_EMU
    (void)edge;
    if (threadIdx.x == 0) {
        unsigned long long* bar = M.mbar + slot;
        ark_mbar_expect_tx(bar, 5u * NCOL * (unsigned)sizeof(double));
        ark_tma_load_4d(M.UR + slot * 5 * NCOL, M.tmap, M.tx, M.ty, k + ARK_NG, 0, bar);
    }
#else
    for (int e = 0; e < (edge ? 2 : 1); ++e) {
        const double* c = (e ? M.Ucol2 : M.Ucol) + M.pstride * (long long)k;
        double* d = M.UR + slot * 5 * NCOL + (e ? M.tc2 : M.tc);
        for (int f = 0; f < 5; ++f) d[f * NCOL] = c[f * M.fs];
    }
#endif
}

template <bool VISC, int TX, int TY>
ARK_DEV void ark_ring_wait(ArkMarch<VISC, TX, TY>& M, int slot) {
#ifndef ARK_HOST_EMU
    ark_mbar_wait(M.mbar + slot, (M.phase >> slot) & 1u);
    M.phase ^= 1u << slot;
#else
    (void)M; (void)slot;
#endif
}

template <bool VISC, int TX, int TY>
ARK_DEV void ark_store_prims(const ArkMarch<VISC, TX, TY>& M, int slot, int tc, const ArkPrim& w) {
    using C = ArkStepCfg<3, VISC, TX, TY>;
    double* p = M.PB + slot * C::NP * C::NCOL + tc;
    p[0] = w.rho; p[C::NCOL] = w.u; p[2 * C::NCOL] = w.v; p[3 * C::NCOL] = w.w;
    p[4 * C::NCOL] = w.p; p[5 * C::NCOL] = w.rc; p[6 * C::NCOL] = w.irc;
    if (VISC) p[7 * C::NCOL] = w.T;
}

template <bool VISC, int TX, int TY>
ARK_DEV ArkPrim ark_march_prims(const ArkParams& P, const ArkMarch<VISC, TX, TY>& M, int tc, int slot) {
    constexpr int NCOL = ArkStepCfg<3, VISC, TX, TY>::NCOL;
    const double* u = M.UR + slot * 5 * NCOL + tc;
    return ark_prim_fast(P, u[0], u[NCOL], u[2 * NCOL], u[3 * NCOL], u[4 * NCOL]);
}

template <bool VISC, int TX, int TY, int ROLE, bool STEADY>
ARK_DEV void ark_plane(const ArkParams& P, const ArkStepConst& K, ArkMarch<VISC, TX, TY>& M, const int q) {
    using C = ArkStepCfg<3, VISC, TX, TY>;
    constexpr int RX = C::RX, NCOL = C::NCOL, NP = C::NP;
    const int tc = M.tc;
    const double lam = K.lam;
    const bool do_update = STEADY || (q >= M.k0 && q < M.k1);     // plane q is an output plane of this chunk
    const bool has_zlo = STEADY || q >= M.k0;                     // face (q-1|q) bounds an output plane
    const bool completes = STEADY || q > M.k0;                    // plane q-1 is completed and stored here

    // ---------------- S1: prefetch plane q+2, primitives of plane q+1 (own column)
    if (STEADY || q + 2 <= M.k1 + 1) ark_ring_issue(M, q + 2, M.unn, ROLE == 1);
    ark_ring_wait(M, M.un);                                       // plane q+1 of the own row(s) has landed
    const ArkPrim wn = ark_march_prims(P, M, tc, M.un);
    ark_store_prims(M, M.pn, tc, wn);
    if (ROLE == 1) ark_store_prims(M, M.pn, M.tc2, ark_march_prims(P, M, M.tc2, M.un));
    // (no barrier: S2 reads the neighbours' primitives of plane q, written one iteration ago)

    // ---------------- S2: acoustic faces of plane q, centred velocity differences
    const double* pq = M.PB + M.pc * NP * NCOL + tc;
    const double rho = M.wc.rho, u = M.wc.u, v = M.wc.v, w = M.wc.w, p = M.wc.p, rc = M.wc.rc, irc = M.wc.irc;
    ArkFace fy;
    {
        const double* n = pq - RX;
        fy = ark_face(P.theta, P.D.gh[1], n[0], n[2 * NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], rho, v, p, rc, irc);
        M.FB[2 * NCOL + tc] = fy.us; M.FB[3 * NCOL + tc] = fy.pi;
    }
    if (ROLE == 1 && M.top) {                                     // low-y face of the edge row RY-1 (own cell | edge cell)
        const double* e = pq + RX;
        const ArkFace f2 = ark_face(P.theta, P.D.gh[1], rho, v, p, rc, irc, e[0], e[2 * NCOL], e[4 * NCOL], e[5 * NCOL], e[6 * NCOL]);
        M.FB[2 * NCOL + M.tc2] = f2.us; M.FB[3 * NCOL + M.tc2] = f2.pi;
    }
    ArkFace fx, zhi;
    double dxu = 0, dxv = 0, dxw = 0, dyu = 0, dyv = 0, dyw = 0, dzu = 0, dzv = 0, dzw = 0;
    {
        const double* n = pq - 1;
        fx = ark_face(P.theta, P.D.gh[0], n[0], n[NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], rho, u, p, rc, irc);
        if (!ARK_XSHFL(RX)) { M.FB[0 * NCOL + tc] = fx.us; M.FB[1 * NCOL + tc] = fx.pi; }
        zhi = ark_face(P.theta, P.D.gh[2], rho, w, p, rc, irc, wn.rho, wn.w, wn.p, wn.rc, wn.irc);
        if (VISC) {
            // un-normalised centred differences q(+1) - q(-1)
            dxu = pq[NCOL + 1] - pq[NCOL - 1];
            dxv = pq[2 * NCOL + 1] - pq[2 * NCOL - 1];
            dxw = pq[3 * NCOL + 1] - pq[3 * NCOL - 1];
            dyu = pq[NCOL + RX] - pq[NCOL - RX];
            dyv = pq[2 * NCOL + RX] - pq[2 * NCOL - RX];
            dyw = pq[3 * NCOL + RX] - pq[3 * NCOL - RX];
            dzu = wn.u - M.wm[0]; dzv = wn.v - M.wm[1]; dzw = wn.w - M.wm[2];
            if (!ARK_XSHFL(RX)) { M.GB[0 * NCOL + tc] = dyu; M.GB[1 * NCOL + tc] = dyv; M.GB[2 * NCOL + tc] = dzu; }
            M.GB[3 * NCOL + tc] = dzw;
            M.GB[4 * NCOL + tc] = dxv; M.GB[5 * NCOL + tc] = dxu; M.GB[6 * NCOL + tc] = dzv;
        }
    }
    __syncthreads();                                              // (B) faces, differences (and prims q+1) visible

    // ---------------- S3: acoustic update U~(q), PAPER.md:158-160 (+ reading A3 for the energy)
    double Uc[5] = {0, 0, 0, 0, 0}, Ut[5] = {0, 0, 0, 0, 0};
    double usxh = 0, pixh = 0, usyh = 0, piyh = 0, Six = 0, Siy = 0, Siz = 0;
    ArkVisc vx = {0, 0, 0, 0}, vy = {0, 0, 0, 0}, vz = {0, 0, 0, 0};
    {
        const double* uc = M.UR + M.uq * 5 * NCOL + tc;
        Uc[0] = rho; Uc[1] = uc[NCOL]; Uc[2] = uc[2 * NCOL]; Uc[3] = uc[3 * NCOL]; Uc[4] = uc[4 * NCOL];
        if (ARK_XSHFL(RX)) { usxh = ark_from_right(fx.us); pixh = ark_from_right(fx.pi); }
        else               { usxh = M.FB[0 * NCOL + tc + 1]; pixh = M.FB[1 * NCOL + tc + 1]; }
        usyh = M.FB[2 * NCOL + tc + RX]; piyh = M.FB[3 * NCOL + tc + RX];
        // S_i = (S_low + S_high)/2; the high face's S is recomputed exactly as its owner computes it
        if (P.D.g_on[0]) Six = 0.5 * (fx.S + (0.5 * P.D.gh[0]) * (rho + pq[1]));
        if (P.D.g_on[1]) Siy = 0.5 * (fy.S + (0.5 * P.D.gh[1]) * (rho + pq[RX]));
        Siz = 0.5 * (zhi.S + M.zlo.S);
        const double sdu = (usxh - fx.us) + (usyh - fy.us) + (zhi.us - M.zlo.us);
        const double sdpu = (pixh * usxh - fx.pi * fx.us) + (piyh * usyh - fy.pi * fy.us) + (zhi.pi * zhi.us - M.zlo.pi * M.zlo.us);
        const double iLt = ark_rcp(1.0 + lam * sdu);
        Ut[0] = Uc[0] * iLt;
        Ut[1] = (Uc[1] - lam * (pixh - fx.pi) + lam * Six) * iLt;
        Ut[2] = (Uc[2] - lam * (piyh - fy.pi) + lam * Siy) * iLt;
        Ut[3] = (Uc[3] - lam * (zhi.pi - M.zlo.pi) + lam * Siz) * iLt;
        Ut[4] = (Uc[4] - lam * sdpu) * iLt;
        double* tb = M.TB + M.tq * 5 * NCOL + tc;
        tb[0] = Ut[0]; tb[NCOL] = Ut[1]; tb[2 * NCOL] = Ut[2]; tb[3 * NCOL] = Ut[3]; tb[4 * NCOL] = Ut[4];

        // viscous / heat fluxes through the low x, low y faces of plane q and the z face (q-1 | q)
        if (VISC) {
            const double Tc = M.wc.T;
            if (do_update) {
                if (ROLE == 2) {   // face (ci-1 | ci), normal x, transverse a = y, b = z
                    const double* L = pq - 1;
                    const double uL = L[NCOL], vL = L[2 * NCOL], wL = L[3 * NCOL], TL = L[7 * NCOL];
                    const int l = tc - 1;
                    double g0, g1, g2, g3;       // dyu, dyv, dzu, dzw of the left cell
                    if (ARK_XSHFL(RX)) { g0 = ark_from_left(dyu); g1 = ark_from_left(dyv); g2 = ark_from_left(dzu); g3 = ark_from_left(dzw); }
                    else { g0 = M.GB[0 * NCOL + l]; g1 = M.GB[1 * NCOL + l]; g2 = M.GB[2 * NCOL + l]; g3 = M.GB[3 * NCOL + l]; }
                    vx = ark_visc_face(P.D.KV, u - uL, v - vL, w - wL, g0 + dyu, g1 + dyv, g2 + dzu, g3 + dzw,
                                       uL + u, vL + v, wL + w, Tc - TL);
                    if (!ARK_XSHFL(RX)) {
                        M.VB[0 * NCOL + tc] = vx.t0; M.VB[1 * NCOL + tc] = vx.t1; M.VB[2 * NCOL + tc] = vx.t2; M.VB[3 * NCOL + tc] = vx.fe;
                    }
                }
                {                  // face (cj-1 | cj), normal y, transverse a = x, b = z (row 1 computes it for nobody)
                    const double* L = pq - RX;
                    const double uL = L[NCOL], vL = L[2 * NCOL], wL = L[3 * NCOL], TL = L[7 * NCOL];
                    const int l = tc - RX;
                    vy = ark_visc_face(P.D.KV, v - vL, u - uL, w - wL, M.GB[4 * NCOL + l] + dxv, M.GB[5 * NCOL + l] + dxu,
                                       M.GB[6 * NCOL + l] + dzv, M.GB[3 * NCOL + l] + dzw, vL + v, uL + u, wL + w, Tc - TL);
                    // stored as (tau_yx, tau_yy, tau_yz, fe): component order x,y,z
                    M.VB[4 * NCOL + tc] = vy.t1; M.VB[5 * NCOL + tc] = vy.t0; M.VB[6 * NCOL + tc] = vy.t2; M.VB[7 * NCOL + tc] = vy.fe;
                }
            }
            if (ROLE == 2) {
                if (has_zlo) {     // face (q-1 | q), normal z, transverse a = x, b = y
                    const double um = M.wm[0], vm = M.wm[1], wm = M.wm[2], Tm = M.wm[3];
                    vz = ark_visc_face(P.D.KV, w - wm, u - um, v - vm, M.gpz[0] + dxw, M.gpz[1] + dxu, M.gpz[2] + dyw, M.gpz[3] + dyv,
                                       wm + w, um + u, vm + v, Tc - Tm);
                }
                M.gpz[0] = dxw; M.gpz[1] = dxu; M.gpz[2] = dyw; M.gpz[3] = dyv;
            }
        }
    }
    __syncthreads();                                              // (C) U~(q) and viscous fluxes visible

    // ---------------- S4: transport + update
    if (ROLE == 2) {
        const double* Tq = M.TB + M.tq * 5 * NCOL;
        double Gz[5] = {0, 0, 0, 0, 0};       // full flux through the z face (q-1|q)
        double mzf = 0.0;
        if (has_zlo) {
            // upwind on u* (reading A10): U~(q-1) or U~(q) of the own column, both in the TB ring
            const double* Tu = M.TB + (ark_nonneg(M.zlo.us) ? (M.tq ^ 1) : M.tq) * 5 * NCOL + tc;
            const double zus = M.zlo.us, zpi = M.zlo.pi;
            Gz[0] = Tu[0] * zus;
            Gz[1] = Tu[NCOL] * zus;
            Gz[2] = Tu[2 * NCOL] * zus;
            Gz[3] = Tu[3 * NCOL] * zus + zpi;
            Gz[4] = (Tu[4 * NCOL] + zpi) * zus;
            mzf = Gz[0];
            if (VISC) { Gz[1] -= vz.t1; Gz[2] -= vz.t2; Gz[3] -= vz.t0; Gz[4] -= vz.fe; }
            if (completes) {
                // complete and store U^{n+1}(q-1):  acc - lam * G_z(high) + gravity work of the high face
                double out[5];
                for (int f = 0; f < 5; ++f) out[f] = M.acc[f] - lam * Gz[f];
                if (P.D.g_on[2]) out[4] += K.dt * P.g[2] * ark_neg_part(mzf);
                if (M.inU) {
                    double* __restrict__ c = M.Ocur;             // plane q-1 of the own column
                    c[0] = out[0];
                    c[M.fs] = out[1];
                    c[2 * M.fs] = out[2];
                    c[3 * M.fs] = out[3];
                    c[4 * M.fs] = out[4];
                }
                if (M.want_rate) {
                    const ark_u64 r = ark_rate_epilogue(P, 3, out[0], out[1], out[2], out[3], out[4], P.D.inv_h, P.D.dcoef);
                    M.rate_max = ark_umax(M.rate_max, M.inU ? r : 0ULL);
                }
            }
        }
        if (do_update) {
            // in-plane faces of plane q: dG = sum_d (F_d+ - F_d-)
            double dG[5];
            double work = 0.0;
            ark_transport_axis<3, 1>(Tq, NCOL, tc, 1, fx.us, fx.pi, usxh, pixh, P.D.g_on[0], P.g[0], dG, work, true);
            ark_transport_axis<3, 2>(Tq, NCOL, tc, RX, fy.us, fy.pi, usyh, piyh, P.D.g_on[1], P.g[1], dG, work, false);
            if (VISC) {
                double h0, h1, h2, h3;           // viscous flux through the high-x face = the right cell's low-x face
                if (ARK_XSHFL(RX)) { h0 = ark_from_right(vx.t0); h1 = ark_from_right(vx.t1); h2 = ark_from_right(vx.t2); h3 = ark_from_right(vx.fe); }
                else { h0 = M.VB[0 * NCOL + tc + 1]; h1 = M.VB[1 * NCOL + tc + 1]; h2 = M.VB[2 * NCOL + tc + 1]; h3 = M.VB[3 * NCOL + tc + 1]; }
                dG[1] -= (h0 - vx.t0) + (M.VB[4 * NCOL + tc + RX] - vy.t1);
                dG[2] -= (h1 - vx.t1) + (M.VB[5 * NCOL + tc + RX] - vy.t0);
                dG[3] -= (h2 - vx.t2) + (M.VB[6 * NCOL + tc + RX] - vy.t2);
                dG[4] -= (h3 - vx.fe) + (M.VB[7 * NCOL + tc + RX] - vy.fe);
            }
            // low z face enters with +lam*G_z and the gravity work dt g_z max(m,0); the source lam*S_i
            M.acc[0] = (Uc[0] - lam * dG[0]) + lam * Gz[0];
            M.acc[1] = (Uc[1] - lam * dG[1] + lam * Six) + lam * Gz[1];
            M.acc[2] = (Uc[2] - lam * dG[2] + lam * Siy) + lam * Gz[2];
            M.acc[3] = (Uc[3] - lam * dG[3]) + lam * Gz[3];
            M.acc[4] = (Uc[4] - lam * dG[4] + K.dt * work) + lam * Gz[4];
            if (P.D.g_on[2]) {
                M.acc[3] += lam * Siz;
                M.acc[4] += K.dt * P.g[2] * ark_pos_part(mzf);
            }
        }
    }
    // rotate the rings; the output pointer follows plane q (kept in registers: recomputing it from the block and
    // thread indices costs ~40 integer instructions per plane)
    if (ROLE == 2) {
        M.Ocur += M.pstride;
#ifndef ARK_HOST_EMU
        asm volatile("" : "+l"(M.Ocur));
#endif
    }
    M.zlo = zhi;
    if (VISC) { M.wm[0] = u; M.wm[1] = v; M.wm[2] = w; M.wm[3] = M.wc.T; }
    M.wc = wn;
    { const int s = M.uq; M.uq = M.un; M.un = M.unn; M.unn = s; }
    { const int s = M.pc; M.pc = M.pn; M.pn = s; }
    M.tq ^= 1;
}

template <bool VISC, int TX, int TY, int ROLE>
ARK_DEV void ark_march(const ArkParams& P, const ArkStepConst& K, ArkMarch<VISC, TX, TY>& M) {
    int q = M.k0 - 1;
    for (; q <= M.k0; ++q) ark_plane<VISC, TX, TY, ROLE, false>(P, K, M, q);    // k0-1, k0
    for (; q < M.k1; ++q) ark_plane<VISC, TX, TY, ROLE, true>(P, K, M, q);      // k0+1 .. k1-1
    for (; q <= M.k1; ++q) ark_plane<VISC, TX, TY, ROLE, false>(P, K, M, q);    // k1
}

template <bool VISC, int TX, int TY>
ARK_DEV void ark_step3d(const ArkParams& P, const double* __restrict__ Uin, double* __restrict__ Uout, double dt_value,
                        const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk, double* smem,
                        const void* tmap) {
    using C = ArkStepCfg<3, VISC, TX, TY>;
    constexpr int RX = C::RX, RY = C::RY, NCOL = C::NCOL, NP = C::NP;
    ArkMarch<VISC, TX, TY> M;
    M.UR = smem;                                      // [3][5][NCOL]
    M.PB = smem + 15 * NCOL;                          // [2][NP][NCOL]
    M.FB = M.PB + 2 * NP * NCOL;                      // [4][NCOL]: usx,pix,usy,piy (low faces of plane q)
    M.TB = M.FB + 4 * NCOL;                           // [2][5][NCOL]: U~ of planes q-1, q
    M.GB = M.TB + 10 * NCOL;                          // [7][NCOL]: dyu,dyv,dzu,dzw,dxv,dxu,dzv (VISC)
    M.VB = M.GB + (VISC ? 7 : 0) * NCOL;              // [8][NCOL]: viscous low-face fluxes x(4), y(4) (VISC)
    ark_u64* red = (ark_u64*)(M.VB + (VISC ? 8 : 0) * NCOL);   // [32]
    unsigned long long* mbars = red + 32;             // [3]

    // thread -> column of rows 1..RY-2 (one warp per row when RX == 32)
    const int t = threadIdx.x;
    const int tc = (t < C::NTHR ? t : C::NTHR - 1) + RX;
    const int ci = tc % RX, cj = tc / RX;
    const int gi = blockIdx.x * TX - 2 + ci, gj = blockIdx.y * TY - 2 + cj;   // interior-based cell coordinates
    // columns beyond the padded array (ragged tiles) load a valid cell; nobody consumes their results
    const int li = gi < P.nx + 2 ? gi : P.nx + 1;
    const int lj = gj < P.ny + 2 ? gj : P.ny + 1;
    M.tc = tc;
    M.k0 = blockIdx.z * zchunk;
    M.k1 = M.k0 + zchunk < P.nz ? M.k0 + zchunk : P.nz;
    const bool rowU = cj >= 2 && cj <= RY - 3;      // tile rows; the others (1, RY-2) are the ring
    M.inU = t < C::NTHR && rowU && ci >= 2 && ci < 2 + TX && gi < P.nx && gj < P.ny;   // stores / rate only
    M.want_rate = rate_scratch != nullptr;
    // ring rows also serve the edge row next to them (row 0 below row 1, row RY-1 above row RY-2)
    M.top = cj == RY - 2;
    M.tc2 = M.top ? tc + RX : tc - RX;
    const int gj2 = M.top ? gj + 1 : gj - 1;
    const int lj2 = gj2 < P.ny + 2 ? gj2 : P.ny + 1;

    const ArkStepConst K = ark_step_const(P, dt_value, dt_dev);
    const long long colbase = (long long)(li + ARK_XOFF) + (long long)P.px * (long long)(lj + ARK_NG);
    M.pstride = (long long)P.px * P.py;
    M.Ucol = Uin + colbase + M.pstride * (long long)P.offz;    // plane 0 of this column
    M.Ucol2 = M.Ucol + (long long)P.px * (long long)(lj2 - lj);
    M.Ocur = Uout + colbase + M.pstride * (long long)(P.offz + M.k0 - 2);   // plane q-1 at q = k0-1
    M.fs = P.fstride;
    M.tmap = tmap;
    M.tx = (int)(blockIdx.x * TX) - 2 + ARK_XOFF;
    M.ty = (int)(blockIdx.y * TY) - 2 + ARK_NG;
    M.mbar = mbars;
    M.phase = 0;
#ifndef ARK_HOST_EMU
    if (t == 0) {
        for (int s3 = 0; s3 < 3; ++s3) ark_mbar_init(M.mbar + s3, 1);
        ark_mbar_fence_init();
    }
    __syncthreads();
#endif

    // ring slots at q = k0-1: UR planes (k0-2,) k0-1, k0, k0+1 -> slots (0,) 1, 2, 0
    M.uq = 1; M.un = 2; M.unn = 0;
    M.pc = 0; M.pn = 1;
    M.tq = 0;

    // ---- prologue: planes k0-2, k0-1 (and k0 in flight)
    for (int s3 = 0; s3 < 3; ++s3) ark_ring_issue(M, M.k0 - 2 + s3, s3, !rowU);
    ark_ring_wait(M, 0);
    ark_ring_wait(M, 1);
    {
        const ArkPrim wm = ark_march_prims(P, M, tc, 0);
        const ArkPrim wc0 = ark_march_prims(P, M, tc, 1);
        M.wm[0] = wm.u; M.wm[1] = wm.v; M.wm[2] = wm.w; M.wm[3] = wm.T;
        M.wc = wc0;
        ark_store_prims(M, M.pc, tc, wc0);
        if (!rowU) ark_store_prims(M, M.pc, M.tc2, ark_march_prims(P, M, M.tc2, 1));
        M.zlo = ark_face(P.theta, P.D.gh[2], wm.rho, wm.w, wm.p, wm.rc, wm.irc, wc0.rho, wc0.w, wc0.p, wc0.rc, wc0.irc);
    }
    for (int f = 0; f < 5; ++f) M.acc[f] = 0.0;
    for (int f = 0; f < 4; ++f) M.gpz[f] = 0.0;
    M.rate_max = 0;
    __syncthreads();                                  // primitives of plane k0-1 visible to the neighbours

    if (rowU) ark_march<VISC, TX, TY, 2>(P, K, M);
    else      ark_march<VISC, TX, TY, 1>(P, K, M);

    if (rate_scratch) {
        // block-wide max of the rate bit patterns -> one double per block
        ark_u64 m = M.rate_max;
#ifndef ARK_HOST_EMU
        for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        const int lane = t & 31, wid = t >> 5;
        if (lane == 0) red[wid] = m;
        __syncthreads();
        if (wid == 0) {
            m = lane < (int)(C::NT / 32) ? red[lane] : 0;
            for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        }
#else
        m = ark_emu_block_umax(m);
        (void)red;
#endif
        if (t == 0) rate_scratch[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = ark_rate_from_bits(m);
    }
}

// ------------------------------------------------------------------------------------------------------------
// 2D body: one plane, same phases, direct loads
// ------------------------------------------------------------------------------------------------------------
template <bool VISC, int TX, int TY>
ARK_DEV void ark_step2d(const ArkParams& P, const double* __restrict__ Uin, double* __restrict__ Uout, double dt_value,
                        const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, double* smem) {
    using C = ArkStepCfg<2, VISC, TX, TY>;
    constexpr int RX = C::RX, RY = C::RY, NCOL = C::NCOL, NP = C::NP;
    double* PB = smem;                                // [NP][NCOL]
    double* FB = PB + NP * NCOL;                      // [6][NCOL]
    double* TB = FB + 6 * NCOL;                       // [5][NCOL] (component 3 unused)
    double* GB = TB + 5 * NCOL;                       // [7][NCOL] (VISC)
    double* VB = GB + (VISC ? 7 : 0) * NCOL;          // [8][NCOL] (VISC)
    ark_u64* red = (ark_u64*)(VB + (VISC ? 8 : 0) * NCOL);

    const int t = threadIdx.x;
    const int tc = t < NCOL ? t : NCOL - 1;
    const int ci = tc % RX, cj = tc / RX;
    const int gi = blockIdx.x * TX - 2 + ci, gj = blockIdx.y * TY - 2 + cj;
    const int li = gi < P.nx + 2 ? gi : P.nx + 1;
    const int lj = gj < P.ny + 2 ? gj : P.ny + 1;
    const bool rowF = cj >= 1;
    const bool rowA = cj >= 1 && cj <= RY - 2;
    const bool rowU = cj >= 2 && cj <= RY - 3;
    const bool rowVy = cj >= 2 && cj <= RY - 2;
    const bool inU = t < NCOL && rowU && ci >= 2 && ci < 2 + TX && gi < P.nx && gj < P.ny;

    const ArkStepConst K = ark_step_const(P, dt_value, dt_dev);
    const double lam = K.lam;
    const long long colbase = (long long)(li + ARK_XOFF) + (long long)P.px * (long long)(lj + ARK_NG);
    const long long fs = P.fstride;

    // S1
    double Uc[5];
    Uc[0] = Uin[colbase]; Uc[1] = Uin[colbase + fs]; Uc[2] = Uin[colbase + 2 * fs]; Uc[3] = 0.0; Uc[4] = Uin[colbase + 3 * fs];
    const ArkPrim wc = ark_prim_fast(P, Uc[0], Uc[1], Uc[2], 0.0, Uc[4]);
    {
        double* p = PB + tc;
        p[0] = wc.rho; p[NCOL] = wc.u; p[2 * NCOL] = wc.v; p[4 * NCOL] = wc.p; p[5 * NCOL] = wc.rc; p[6 * NCOL] = wc.irc;
        if (VISC) p[7 * NCOL] = wc.T;
    }
    __syncthreads();
    // S2
    const double* pq = PB + tc;
    ArkFace fx = {0, 0, 0}, fy = {0, 0, 0};
    double dxu = 0, dxv = 0, dyu = 0, dyv = 0;
    if (rowF) {
        {
            const double* n = pq - RX;
            fy = ark_face(P.theta, P.D.gh[1], n[0], n[2 * NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], wc.rho, wc.v, wc.p, wc.rc, wc.irc);
            FB[2 * NCOL + tc] = fy.us; FB[3 * NCOL + tc] = fy.pi;
            if (P.D.g_on[1]) FB[5 * NCOL + tc] = fy.S;
        }
        if (rowA) {
            const double* n = pq - 1;
            fx = ark_face(P.theta, P.D.gh[0], n[0], n[NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], wc.rho, wc.u, wc.p, wc.rc, wc.irc);
            FB[0 * NCOL + tc] = fx.us; FB[1 * NCOL + tc] = fx.pi;
            if (P.D.g_on[0]) FB[4 * NCOL + tc] = fx.S;
            if (VISC) {
                dxu = pq[NCOL + 1] - pq[NCOL - 1];
                dxv = pq[2 * NCOL + 1] - pq[2 * NCOL - 1];
                dyu = pq[NCOL + RX] - pq[NCOL - RX];
                dyv = pq[2 * NCOL + RX] - pq[2 * NCOL - RX];
                GB[0 * NCOL + tc] = dyu; GB[1 * NCOL + tc] = dyv; GB[4 * NCOL + tc] = dxv; GB[5 * NCOL + tc] = dxu;
            }
        }
    }
    __syncthreads();
    // S3
    double usxh = 0, pixh = 0, usyh = 0, piyh = 0, Six = 0, Siy = 0;
    ArkVisc vx = {0, 0, 0, 0}, vy = {0, 0, 0, 0};
    if (rowA) {
        usxh = FB[0 * NCOL + tc + 1]; pixh = FB[1 * NCOL + tc + 1];
        usyh = FB[2 * NCOL + tc + RX]; piyh = FB[3 * NCOL + tc + RX];
        if (P.D.g_on[0]) Six = 0.5 * (fx.S + FB[4 * NCOL + tc + 1]);
        if (P.D.g_on[1]) Siy = 0.5 * (fy.S + FB[5 * NCOL + tc + RX]);
        const double sdu = (usxh - fx.us) + (usyh - fy.us);
        const double sdpu = (pixh * usxh - fx.pi * fx.us) + (piyh * usyh - fy.pi * fy.us);
        const double iLt = ark_rcp(1.0 + lam * sdu);
        double* tb = TB + tc;
        tb[0] = Uc[0] * iLt;
        tb[NCOL] = (Uc[1] - lam * (pixh - fx.pi) + lam * Six) * iLt;
        tb[2 * NCOL] = (Uc[2] - lam * (piyh - fy.pi) + lam * Siy) * iLt;
        tb[4 * NCOL] = (Uc[4] - lam * sdpu) * iLt;
    }
    if (VISC && rowVy) {
        if (rowU) {
            const double* L = pq - 1;
            const double uL = L[NCOL], vL = L[2 * NCOL], TL = L[7 * NCOL];
            const int l = tc - 1;
            vx = ark_visc_face(P.D.KV, wc.u - uL, wc.v - vL, 0.0, GB[0 * NCOL + l] + dyu, GB[1 * NCOL + l] + dyv, 0.0, 0.0,
                               uL + wc.u, vL + wc.v, 0.0, wc.T - TL);
            VB[0 * NCOL + tc] = vx.t0; VB[1 * NCOL + tc] = vx.t1; VB[3 * NCOL + tc] = vx.fe;
        }
        {
            const double* L = pq - RX;
            const double uL = L[NCOL], vL = L[2 * NCOL], TL = L[7 * NCOL];
            const int l = tc - RX;
            vy = ark_visc_face(P.D.KV, wc.v - vL, wc.u - uL, 0.0, GB[4 * NCOL + l] + dxv, GB[5 * NCOL + l] + dxu, 0.0, 0.0,
                               vL + wc.v, uL + wc.u, 0.0, wc.T - TL);
            VB[4 * NCOL + tc] = vy.t1; VB[5 * NCOL + tc] = vy.t0; VB[7 * NCOL + tc] = vy.fe;
        }
    }
    __syncthreads();
    // S4
    ark_u64 rate_max = 0;
    if (rowU) {
        double dG[5];
        double work = 0.0;
        ark_transport_axis<2, 1>(TB, NCOL, tc, 1, fx.us, fx.pi, usxh, pixh, P.D.g_on[0], P.g[0], dG, work, true);
        ark_transport_axis<2, 2>(TB, NCOL, tc, RX, fy.us, fy.pi, usyh, piyh, P.D.g_on[1], P.g[1], dG, work, false);
        if (VISC) {
            dG[1] -= (VB[0 * NCOL + tc + 1] - vx.t0) + (VB[4 * NCOL + tc + RX] - vy.t1);
            dG[2] -= (VB[1 * NCOL + tc + 1] - vx.t1) + (VB[5 * NCOL + tc + RX] - vy.t0);
            dG[4] -= (VB[3 * NCOL + tc + 1] - vx.fe) + (VB[7 * NCOL + tc + RX] - vy.fe);
        }
        const double n0 = Uc[0] - lam * dG[0];
        const double n1 = Uc[1] - lam * dG[1] + lam * Six;
        const double n2 = Uc[2] - lam * dG[2] + lam * Siy;
        const double n4 = Uc[4] - lam * dG[4] + K.dt * work;
        if (inU) {
            Uout[colbase] = n0; Uout[colbase + fs] = n1; Uout[colbase + 2 * fs] = n2; Uout[colbase + 3 * fs] = n4;
            if (rate_scratch) rate_max = ark_rate_epilogue(P, 2, n0, n1, n2, 0.0, n4, P.D.inv_h, P.D.dcoef);
        }
    }
    if (rate_scratch) {
        ark_u64 m = rate_max;
#ifndef ARK_HOST_EMU
        for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        const int lane = t & 31, wid = t >> 5;
        if (lane == 0) red[wid] = m;
        __syncthreads();
        if (wid == 0) {
            m = lane < (int)(C::NT / 32) ? red[lane] : 0;
            for (int o = 16; o > 0; o >>= 1) m = ark_umax(m, __shfl_xor_sync(0xffffffffu, m, o));
        }
#else
        m = ark_emu_block_umax(m);
        (void)red;
#endif
        if (t == 0) rate_scratch[blockIdx.x + gridDim.x * blockIdx.y] = ark_rate_from_bits(m);
    }
}

// the tensor map of the input state rides in the kernel parameter bank (3D; the 2D kernels ignore it)
#ifndef ARK_HOST_EMU
#define ARK_TMAP_PARAM , const __grid_constant__ CUtensorMap tmap
#define ARK_TMAP_ARG &tmap
#else
#define ARK_TMAP_PARAM
#define ARK_TMAP_ARG nullptr
#endif

template <int NDIM, bool VISC, int TX, int TY>
ARK_GLOBAL void
#ifndef ARK_HOST_EMU
__launch_bounds__(ArkStepCfg<NDIM, VISC, TX, TY>::NT, NDIM == 3 ? 1 : 2)   // 2D: two single-plane blocks per SM overlap their barriers
#endif
ark_k_step(const ArkParams P, const double* __restrict__ Uin, double* __restrict__ Uout,
           double dt_value, const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk ARK_TMAP_PARAM) {
    ARK_DYN_SMEM(smem);
    if (NDIM == 3) ark_step3d<VISC, TX, TY>(P, Uin, Uout, dt_value, dt_dev, rate_scratch, zchunk, smem, ARK_TMAP_ARG);
    else           ark_step2d<VISC, TX, TY>(P, Uin, Uout, dt_value, dt_dev, rate_scratch, smem);
}
