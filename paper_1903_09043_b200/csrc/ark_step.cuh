// ark_step.cuh -- helpers shared by the fused step kernels and the 2D kernel (acoustic + transport + dissipative +
// update + CFL epilogue in one launch).
//
// One launch advances U^n -> U^{n+1}: every conserved field is read once and written once (64 B per cell update in
// 2D, 80 B in 3D: ark_step3d.cuh); all face quantities, velocity gradients and the intermediate state U~ live in
// registers / shared memory only.
//
// 2D (nz == 1): a block owns a TX x TY tile of cells plus a 2-cell halo (region RX x RY = (TX+4) x (TY+4)), one thread
// per region cell, direct loads (the 2D configurations are L2-resident, launch / latency-bound), three barriers:
//   S1 primitives -> PB | S2 acoustic faces x-, y- (PAPER.md:152, 218-222), centred velocity differences -> FB, GB |
//   S3 acoustic update U~ -> TB, viscous / heat fluxes of the low faces -> VB | S4 transport
//   (upwind on u*), conservative update (eq. 11), store, CFL rate of the new state.
//
// GEN = the general path: an array-valued potential Phi (every face uses
// its own -(Phi_R - Phi_L) instead of g_d h, the gravity work uses the upwind potential) and / or
// the non-conservative energy scheme of Appendix B (P.eform == 1: the energy carries the source
// lam (uS)_i in both sub-steps instead of the gravity work; reading A24).  The standard instantiations carry none of it.
#pragma once
#include "ark_device.cuh"

#define ARK_NPRIM 8   // rho,u,v,w,p,rc,irc,T

template <int NDIM, bool VISC, int TX, int TY>
struct ArkStepCfg {
    static_assert(NDIM == 2, "the 3D kernel has its own configuration (ArkCfg3, ark_step3d.cuh)");
    static constexpr int RX = TX + 4, RY = TY + 4, NCOL = RX * RY;
    static constexpr int NT = ((NCOL + 31) / 32) * 32;               // one thread per region cell
    static constexpr int NP = VISC ? 8 : 7;                          // T only feeds the heat flux
    // shared memory (doubles per column): PB[NP], FB[6], TB[5], GB[7], VB[8] (+ 32 for the reduction)
    static constexpr int PER_COL = NP + 6 + 5 + (VISC ? 15 : 0);
    static constexpr int SMEM_DOUBLES = PER_COL * NCOL + 32;
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
// GEN: the two faces carry their own potential differences gl, gh = -(Phi_R - Phi_L) and work collects
// gl max(m_{d-},0) + gh min(m_{d+},0), to be multiplied by lam; otherwise gl = g_d and work is multiplied by dt.
template <int NDIM, int DN, bool GEN>
ARK_DEV void ark_transport_axis(const double* __restrict__ T, int cs, int tc, int sd, double usl, double pil, double ush,
                                double pih, bool g_on, double gl, double gh, double* dG, double& work, bool first) {
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
    if (g_on) work += GEN ? gl * ark_pos_part(ml) + gh * ark_neg_part(mh) : gl * (ark_pos_part(ml) + ark_neg_part(mh));
}

// ------------------------------------------------------------------------------------------------------------
// 2D body: one plane, same phases, direct loads
// ------------------------------------------------------------------------------------------------------------
template <bool VISC, bool GEN, int TX, int TY>
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

    // GEN: potential of the own cell and of its four neighbours -> -(Phi_R - Phi_L) of the four faces (else g_d h)
    const bool PH = GEN && P.phi != nullptr;
    double ghxl = P.D.gh[0], ghxh = P.D.gh[0], ghyl = P.D.gh[1], ghyh = P.D.gh[1];
    if (PH) {
        const int il = li > -ARK_NG ? li - 1 : li, ir = li < P.nx + 1 ? li + 1 : li;
        const int jb = lj > -ARK_NG ? lj - 1 : lj, ja = lj < P.ny + 1 ? lj + 1 : lj;
        const double* ph = P.phi + ARK_XOFF + (long long)P.px * ARK_NG;
        const double phc = ph[li + (long long)P.px * lj];
        ghxl = ph[il + (long long)P.px * lj] - phc; ghxh = phc - ph[ir + (long long)P.px * lj];
        ghyl = ph[li + (long long)P.px * jb] - phc; ghyh = phc - ph[li + (long long)P.px * ja];
    }
    const bool eformB = GEN && P.eform == 1;

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
            fy = ark_face(P.theta, GEN ? ghyl : P.D.gh[1], n[0], n[2 * NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], wc.rho, wc.v, wc.p, wc.rc, wc.irc);
            FB[2 * NCOL + tc] = fy.us; FB[3 * NCOL + tc] = fy.pi;
            if (P.D.g_on[1]) FB[5 * NCOL + tc] = fy.S;
        }
        if (rowA) {
            const double* n = pq - 1;
            fx = ark_face(P.theta, GEN ? ghxl : P.D.gh[0], n[0], n[NCOL], n[4 * NCOL], n[5 * NCOL], n[6 * NCOL], wc.rho, wc.u, wc.p, wc.rc, wc.irc);
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
    double usxh = 0, pixh = 0, usyh = 0, piyh = 0, Six = 0, Siy = 0, suS = 0;
    ArkVisc vx = {0, 0, 0, 0}, vy = {0, 0, 0, 0};
    if (rowA) {
        usxh = FB[0 * NCOL + tc + 1]; pixh = FB[1 * NCOL + tc + 1];
        usyh = FB[2 * NCOL + tc + RX]; piyh = FB[3 * NCOL + tc + RX];
        double Sxh = 0, Syh = 0;
        if (P.D.g_on[0]) { Sxh = FB[4 * NCOL + tc + 1]; Six = 0.5 * (fx.S + Sxh); }
        if (P.D.g_on[1]) { Syh = FB[5 * NCOL + tc + RX]; Siy = 0.5 * (fy.S + Syh); }
        const double sdu = (usxh - fx.us) + (usyh - fy.us);
        const double sdpu = (pixh * usxh - fx.pi * fx.us) + (piyh * usyh - fy.pi * fy.us);
        const double iLt = ark_rcp(1.0 + lam * sdu);
        double* tb = TB + tc;
        tb[0] = Uc[0] * iLt;
        tb[NCOL] = (Uc[1] - lam * (pixh - fx.pi) + lam * Six) * iLt;
        tb[2 * NCOL] = (Uc[2] - lam * (piyh - fy.pi) + lam * Siy) * iLt;
        if (eformB) {
            // Appendix B (reading A24): (uS)_i = 1/2 (u*_{i+1/2} S_{i+1/2} + u*_{i-1/2} S_{i-1/2}) per axis
            suS = 0.5 * (usxh * Sxh + fx.us * fx.S) + 0.5 * (usyh * Syh + fy.us * fy.S);
            tb[4 * NCOL] = ((Uc[4] + lam * suS) - lam * sdpu) * iLt;
        } else {
            tb[4 * NCOL] = (Uc[4] - lam * sdpu) * iLt;
        }
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
        const bool wk = !eformB;                    // Appendix B replaces the gravity work by lam (uS)_i
        ark_transport_axis<2, 1, GEN>(TB, NCOL, tc, 1, fx.us, fx.pi, usxh, pixh, wk && P.D.g_on[0], GEN ? ghxl : P.g[0], ghxh, dG, work, true);
        ark_transport_axis<2, 2, GEN>(TB, NCOL, tc, RX, fy.us, fy.pi, usyh, piyh, wk && P.D.g_on[1], GEN ? ghyl : P.g[1], ghyh, dG, work, false);
        if (VISC) {
            dG[1] -= (VB[0 * NCOL + tc + 1] - vx.t0) + (VB[4 * NCOL + tc + RX] - vy.t1);
            dG[2] -= (VB[1 * NCOL + tc + 1] - vx.t1) + (VB[5 * NCOL + tc + RX] - vy.t0);
            dG[4] -= (VB[3 * NCOL + tc + 1] - vx.fe) + (VB[7 * NCOL + tc + RX] - vy.fe);
        }
        const double n0 = Uc[0] - lam * dG[0];
        const double n1 = Uc[1] - lam * dG[1] + lam * Six;
        const double n2 = Uc[2] - lam * dG[2] + lam * Siy;
        const double n4 = GEN ? Uc[4] - lam * dG[4] + lam * (eformB ? suS : work) : Uc[4] - lam * dG[4] + K.dt * work;
        if (inU) {
            Uout[colbase] = n0; Uout[colbase + fs] = n1; Uout[colbase + 2 * fs] = n2; Uout[colbase + 3 * fs] = n4;
            // periodic x: the first / last two columns also fill the opposite ghost columns of the new state,
            // so that the next step needs no x ghost-fill launch (as in the 3D kernel)
            const bool perx = P.bc[0][0] == ARK_BCK_PERIODIC, pery = perx && P.bc[1][0] == ARK_BCK_PERIODIC;
            const long long wx = (perx && gi < ARK_NG) ? P.nx : ((perx && gi >= P.nx - ARK_NG) ? -P.nx : 0);
            // (the y ghost rows are only written here when x is periodic too: their corner cells then come from this kernel
            // as well; with walls in x the y sweep of the ghost-fill kernel copies the wall ghosts of the wrapped rows)
            if (wx != 0) { const long long w = colbase + wx; Uout[w] = n0; Uout[w + fs] = n1; Uout[w + 2 * fs] = n2; Uout[w + 3 * fs] = n4; }
            if (pery && (gj < ARK_NG || gj >= P.ny - ARK_NG)) {      // (uniform test first: nothing of this for wall configurations)
                const long long wy = gj < ARK_NG ? (long long)P.px * P.ny : -(long long)P.px * P.ny;
                { const long long w = colbase + wy; Uout[w] = n0; Uout[w + fs] = n1; Uout[w + 2 * fs] = n2; Uout[w + 3 * fs] = n4; }
                if (wx != 0) { const long long w = colbase + wx + wy; Uout[w] = n0; Uout[w + fs] = n1; Uout[w + 2 * fs] = n2; Uout[w + 3 * fs] = n4; }
            }
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

template <int NDIM, bool VISC, bool GEN, int TX, int TY>
ARK_GLOBAL void
#ifndef ARK_HOST_EMU
__launch_bounds__(ArkStepCfg<NDIM, VISC, TX, TY>::NT, 2)   // two single-plane blocks per SM overlap their barriers
#endif
ark_k_step(const ArkParams P, const double* __restrict__ Uin, double* __restrict__ Uout,
           double dt_value, const double* __restrict__ dt_dev, double* __restrict__ rate_scratch) {
    ARK_DYN_SMEM(smem);
    ark_step2d<VISC, GEN, TX, TY>(P, Uin, Uout, dt_value, dt_dev, rate_scratch, smem);
}
