// ark_step.cuh -- the fused full-step kernel (acoustic + transport + dissipative + update + CFL epilogue).
//
// One launch advances U^n -> U^{n+1}: every conserved field is read once and written once
// (80 B per cell update in 3D, 64 B in 2D); all face quantities, velocity gradients and the intermediate
// state U~ live in registers / shared memory only.
//
// Decomposition ("2.5-D marching"): a block owns a TX x TY tile of (x,y) columns plus a 2-cell halo
// (region RX x RY = (TX+4) x (TY+4), one thread per column) and marches along z over a chunk of planes.
// The product build uses TX = 28, so RX = 32: ONE WARP PER REGION ROW.  Every role that depends on the
// row (halo row / ring row / output row) is then warp-uniform -- halo warps skip whole phases instead of
// idling lanes -- and every global load of a warp is one contiguous 256-byte row segment.
//
// Per plane q one iteration does (3 block barriers):
//   S1  primitives of plane q+1 (own column, from registers)           -> smem PB (2-plane ring)
//   --- barrier A
//   S2  acoustic faces x-, y- of plane q (neighbours from PB), z face (q|q+1) from registers   -> smem FB
//       cell-centred velocity differences of plane q (x,y neighbours from PB, z from registers) -> smem GB
//   --- barrier B
//   S3  acoustic update U~(q) on tile + 1 ring       -> smem TB
//       viscous / heat fluxes through the x-, y- faces of plane q      -> smem VB ; z- face in registers
//   --- barrier C
//   S4  transport fluxes (upwind on u*) of the in-plane faces of plane q and of the
//       z face (q-1|q); completes and stores U^{n+1}(q-1); folds the CFL rate of the new state into a
//       per-block maximum (integer max on the bit patterns, NaN-propagating).
// z neighbours of a column stay in the owning thread's registers; only x/y neighbours go through
// shared memory.
#pragma once
#include "ark_device.cuh"

#define ARK_NPRIM 8   // rho,u,v,w,p,rc,irc,T

template <int TX, int TY>
struct ArkStepCfg {
    static constexpr int RX = TX + 4, RY = TY + 4, NCOL = RX * RY;
    static constexpr int NT = ((NCOL + 31) / 32) * 32;
    // shared memory (doubles per column): PB[2][8] FB[6] GB[7] TB[5] VB[8]  (+ 32 for the block reduction)
    static constexpr int PER_COL = 2 * ARK_NPRIM + 6 + 7 + 5 + 8;
    static constexpr int SMEM_DOUBLES = PER_COL * NCOL + 32;
    static constexpr size_t SMEM_BYTES = (size_t)SMEM_DOUBLES * sizeof(double);
};

// cheap two-way selects (fmax/fmin on doubles expand to DSETP + FSEL/SEL + NaN quieting + moves)
ARK_DEV double ark_sel(bool c, double a, double b) { return c ? a : b; }

// Coefficients of the dissipative face flux, precomputed once per thread.
struct ArkViscCoef { double cn, ct, c43, c23t, kh; };

struct ArkVisc { double t0, t1, t2, fe; };

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
// (see ark_rate_bits): one reciprocal and one square root per cell.
ARK_DEV ark_u64 ark_rate_epilogue(const ArkParams& P, int ndim, double rho, double mx, double my, double mz, double E,
                                  double inv_h, double dcoef) {
    const double rinv = 1.0 / rho;
    const double s = (fabs(mx) + fabs(my) + fabs(mz)) * rinv;
    const double ke = 0.5 * (mx * mx + my * my + mz * mz) * rinv;
    const double c = sqrt(P.gamma * (P.gm1 * (E - ke)) * rinv);
    const double r = (s + (double)ndim * c) * inv_h + dcoef * rinv;
    return ark_rate_bits(r) & 0x7fffffffffffffffULL;
}

template <int NDIM, bool VISC, int TX, int TY>
ARK_GLOBAL void
#ifndef ARK_HOST_EMU
__launch_bounds__(ArkStepCfg<TX, TY>::NT, 1)
#endif
ark_k_step(const ArkParams P, const double* __restrict__ Uin, double* __restrict__ Uout,
           double dt_value, const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk) {
    using C = ArkStepCfg<TX, TY>;
    constexpr int RX = C::RX, RY = C::RY, NCOL = C::NCOL;
    constexpr int NF = NDIM == 3 ? 5 : 4;
    constexpr int FE = NF - 1;                        // index of the energy field in HBM
    ARK_DYN_SMEM(smem);
    double* PB = smem;                                // [2][NPRIM][NCOL]
    double* FB = PB + 2 * ARK_NPRIM * NCOL;           // [6][NCOL]: usx,pix,usy,piy,Sx,Sy (low faces of plane q)
    double* GB = FB + 6 * NCOL;                       // [7][NCOL]: dyu,dyv,dzu,dzw,dxv,dxu,dzv (centred differences)
    double* TB = GB + 7 * NCOL;                       // [5][NCOL]: U~(q)
    double* VB = TB + 5 * NCOL;                       // [8][NCOL]: viscous low-face fluxes x(4), y(4)
    ark_u64* red = (ark_u64*)(VB + 8 * NCOL);         // [32]

    const int t = threadIdx.x;
    const bool live = t < NCOL;
    const int tc = live ? t : NCOL - 1;
    const int ci = tc % RX, cj = tc / RX;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int gi = x0 - 2 + ci, gj = y0 - 2 + cj;      // interior-based cell coordinates of this column
    // clamp columns that fall outside the padded array (ragged tiles): they load a valid cell, results unused
    const int li = gi < P.nx + 2 ? gi : P.nx + 1;
    const int lj = gj < P.ny + 2 ? gj : P.ny + 1;

    const int k0 = NDIM == 3 ? blockIdx.z * zchunk : 0;
    const int k1 = NDIM == 3 ? (k0 + zchunk < P.nz ? k0 + zchunk : P.nz) : 1;

    // roles (row conditions are warp-uniform when RX == 32)
    const bool rowA = cj >= 1 && cj <= RY - 2;                           // tile + 1 ring
    const bool rowU = cj >= 2 && cj <= RY - 3;                           // tile
    const bool colA = ci >= 1 && ci <= RX - 2;
    const bool inFx = live && rowA && ci >= 1;                           // owns the low-x face (ci-1 | ci)
    const bool inFy = live && cj >= 1 && colA;                           // owns the low-y face (cj-1 | cj)
    const bool inA = live && rowA && colA && gi <= P.nx && gj <= P.ny;   // acoustic update / centred differences
    const bool inU = live && rowU && ci >= 2 && ci < 2 + TX && gi < P.nx && gj < P.ny;
    const bool inVx = VISC && live && rowU && ci >= 2 && ci <= 2 + TX;
    const bool inVy = VISC && live && cj >= 2 && cj <= 2 + TY && ci >= 2 && ci < 2 + TX;

    const double dt = dt_dev ? dt_dev[1] : dt_value;
    const double inv_h = 1.0 / P.h;
    const double lam = dt / P.h;
    const double ghx = P.g[0] * P.h, ghy = P.g[1] * P.h, ghz = P.g[2] * P.h;
    const bool gx_on = ghx != 0.0, gy_on = ghy != 0.0;
    const int th = P.theta;
    const double dcoef = 2.0 * P.ndim * fmax(4.0 * P.mu / 3.0, P.gm1 * P.kappa) * inv_h * inv_h;
    ArkViscCoef KV;
    KV.cn = P.mu * inv_h; KV.ct = 0.25 * P.mu * inv_h; KV.c43 = (4.0 / 3.0) * P.mu * inv_h;
    KV.c23t = (2.0 / 3.0) * 0.25 * P.mu * inv_h; KV.kh = P.kappa * inv_h;

    const long long colbase = (long long)(li + ARK_XOFF) + (long long)P.px * (long long)(lj + ARK_NG);
    const long long pstride = (long long)P.px * P.py;
    const double* __restrict__ Ucol = Uin + colbase + pstride * (long long)P.offz;   // plane 0 of this column
    double* __restrict__ Ocol = Uout + colbase + pstride * (long long)P.offz;
    const long long fs = P.fstride;

    auto loadU = [&](int k, double* u5) {
        const double* __restrict__ c = Ucol + pstride * (long long)k;
        u5[0] = c[0];
        u5[1] = c[fs];
        u5[2] = c[2 * fs];
        u5[3] = NDIM == 3 ? c[3 * fs] : 0.0;
        u5[4] = c[FE * fs];
    };
    auto pb = [&](int slot, int f, int col) -> double& { return PB[(slot * ARK_NPRIM + f) * NCOL + col]; };
    auto storePrim = [&](int slot, const ArkPrim& w) {
        pb(slot, 0, tc) = w.rho; pb(slot, 1, tc) = w.u; pb(slot, 2, tc) = w.v;
        if (NDIM == 3) pb(slot, 3, tc) = w.w;
        pb(slot, 4, tc) = w.p; pb(slot, 5, tc) = w.rc; pb(slot, 6, tc) = w.irc;
        if (VISC) pb(slot, 7, tc) = w.T;
    };

    ark_u64 rate_max = 0;

    // ---------------------------------------------------------------------------------------------
    // register pipeline along z
    // ---------------------------------------------------------------------------------------------
    double Ucur[5], Unext[5];          // U^n(q), U^n(q+1)
    ArkPrim wc, wn;                    // primitives of own column at q, q+1
    double wmu = 0, wmv = 0, wmw = 0, wmT = 0;  // u,v,w,T of own column at q-1 (viscous z stencil)
    ArkFace zlo = {0, 0, 0}, zhi = {0, 0, 0};   // acoustic z faces (q-1|q), (q|q+1)
    double Utprev[5] = {0, 0, 0, 0, 0};         // U~(q-1) of own column
    double acc[5] = {0, 0, 0, 0, 0};            // U^{n+1}(q-1) minus its high-z flux
    double gpz[4] = {0, 0, 0, 0};               // dxw,dxu,dyw,dyv of own column at q-1 (viscous z face)
    int sc = 0, sn = 1;                // PB slots of planes q, q+1

    if (NDIM == 3) {
        // prologue: planes k0-2 and k0-1
        double Ua[5];
        loadU(k0 - 2, Ua);
        const ArkPrim wm = ark_prim(P, Ua[0], Ua[1], Ua[2], Ua[3], Ua[4]);
        loadU(k0 - 1, Ucur);
        wc = ark_prim(P, Ucur[0], Ucur[1], Ucur[2], Ucur[3], Ucur[4]);
        storePrim(sc, wc);
        zlo = ark_face(th, ghz, wm.rho, wm.w, wm.p, wm.rc, wm.irc, wc.rho, wc.w, wc.p, wc.rc, wc.irc);
        wmu = wm.u; wmv = wm.v; wmw = wm.w; wmT = wm.T;
        loadU(k0, Unext);
    } else {
        loadU(0, Unext);
        wc = ark_prim(P, Unext[0], Unext[1], Unext[2], Unext[3], Unext[4]);
    }

    const int qbeg = NDIM == 3 ? k0 - 1 : 0, qend = NDIM == 3 ? k1 : 0;
    for (int q = qbeg; q <= qend; ++q) {
        // ---------------- S1: primitives of plane q+1 (3D) / plane 0 (2D)
        double Upre[5] = {0, 0, 0, 0, 0};
        if (NDIM == 3) {
            if (q + 2 <= k1 + 1) loadU(q + 2, Upre);           // prefetch, consumed next iteration
            wn = ark_prim(P, Unext[0], Unext[1], Unext[2], Unext[3], Unext[4]);
            storePrim(sn, wn);
        } else {
            for (int f = 0; f < 5; ++f) Ucur[f] = Unext[f];
            wn = wc;
            storePrim(sc, wc);
        }
        __syncthreads();                                       // (A) prims visible

        const bool do_update = NDIM == 2 || (q >= k0 && q < k1);   // plane q is an output plane of this chunk
        // ---------------- S2: acoustic faces of plane q
        ArkFace fx = {0, 0, 0}, fy = {0, 0, 0};
        if (inFx) {
            const int n = tc - 1;
            fx = ark_face(th, ghx, pb(sc, 0, n), pb(sc, 1, n), pb(sc, 4, n), pb(sc, 5, n), pb(sc, 6, n),
                          wc.rho, wc.u, wc.p, wc.rc, wc.irc);
            FB[0 * NCOL + tc] = fx.us; FB[1 * NCOL + tc] = fx.pi;
            if (gx_on) FB[4 * NCOL + tc] = fx.S;
        }
        if (inFy) {
            const int n = tc - RX;
            fy = ark_face(th, ghy, pb(sc, 0, n), pb(sc, 2, n), pb(sc, 4, n), pb(sc, 5, n), pb(sc, 6, n),
                          wc.rho, wc.v, wc.p, wc.rc, wc.irc);
            FB[2 * NCOL + tc] = fy.us; FB[3 * NCOL + tc] = fy.pi;
            if (gy_on) FB[5 * NCOL + tc] = fy.S;
        }
        if (NDIM == 3 && inA)
            zhi = ark_face(th, ghz, wc.rho, wc.w, wc.p, wc.rc, wc.irc, wn.rho, wn.w, wn.p, wn.rc, wn.irc);

        // centred velocity differences of plane q (un-normalised: q(+1) - q(-1)), tile + 1 ring
        double dxu = 0, dxv = 0, dxw = 0, dyu = 0, dyv = 0, dyw = 0, dzu = 0, dzv = 0, dzw = 0;
        if (VISC && inA) {
            dxu = pb(sc, 1, tc + 1) - pb(sc, 1, tc - 1);
            dxv = pb(sc, 2, tc + 1) - pb(sc, 2, tc - 1);
            dyu = pb(sc, 1, tc + RX) - pb(sc, 1, tc - RX);
            dyv = pb(sc, 2, tc + RX) - pb(sc, 2, tc - RX);
            if (NDIM == 3) {
                dxw = pb(sc, 3, tc + 1) - pb(sc, 3, tc - 1);
                dyw = pb(sc, 3, tc + RX) - pb(sc, 3, tc - RX);
                dzu = wn.u - wmu; dzv = wn.v - wmv; dzw = wn.w - wmw;
            }
            GB[0 * NCOL + tc] = dyu; GB[1 * NCOL + tc] = dyv;
            GB[4 * NCOL + tc] = dxv; GB[5 * NCOL + tc] = dxu;
            if (NDIM == 3) { GB[2 * NCOL + tc] = dzu; GB[3 * NCOL + tc] = dzw; GB[6 * NCOL + tc] = dzv; }
        }
        __syncthreads();                                       // (B) faces and differences visible

        // ---------------- S3: acoustic update U~(q), PAPER.md:158-160 (+ reading A3 for the energy)
        double Ut[5] = {0, 0, 0, 0, 0};
        double usxh = 0, pixh = 0, usyh = 0, piyh = 0, Six = 0, Siy = 0, Siz = 0;
        if (inA) {
            usxh = FB[0 * NCOL + tc + 1]; pixh = FB[1 * NCOL + tc + 1];
            usyh = FB[2 * NCOL + tc + RX]; piyh = FB[3 * NCOL + tc + RX];
            if (gx_on) Six = 0.5 * (fx.S + FB[4 * NCOL + tc + 1]);
            if (gy_on) Siy = 0.5 * (fy.S + FB[5 * NCOL + tc + RX]);
            double sdu = (usxh - fx.us) + (usyh - fy.us);
            double sdpu = (pixh * usxh - fx.pi * fx.us) + (piyh * usyh - fy.pi * fy.us);
            if (NDIM == 3) {
                sdu += zhi.us - zlo.us;
                sdpu += zhi.pi * zhi.us - zlo.pi * zlo.us;
                Siz = 0.5 * (zhi.S + zlo.S);
            }
            const double iLt = 1.0 / (1.0 + lam * sdu);
            Ut[0] = Ucur[0] * iLt;
            Ut[1] = (Ucur[1] - lam * (pixh - fx.pi) + lam * Six) * iLt;
            Ut[2] = (Ucur[2] - lam * (piyh - fy.pi) + lam * Siy) * iLt;
            if (NDIM == 3) Ut[3] = (Ucur[3] - lam * (zhi.pi - zlo.pi) + lam * Siz) * iLt;
            Ut[4] = (Ucur[4] - lam * sdpu) * iLt;
            TB[0 * NCOL + tc] = Ut[0]; TB[1 * NCOL + tc] = Ut[1]; TB[2 * NCOL + tc] = Ut[2];
            if (NDIM == 3) TB[3 * NCOL + tc] = Ut[3];
            TB[4 * NCOL + tc] = Ut[4];
        }

        // viscous / heat fluxes through the low x, low y faces of plane q and the z face (q-1 | q)
        ArkVisc vx = {0, 0, 0, 0}, vy = {0, 0, 0, 0}, vz = {0, 0, 0, 0};
        if (VISC) {
            if (do_update && inVx) {   // face (ci-1 | ci), normal x, transverse a = y, b = z
                const int L = tc - 1;
                const double uL = pb(sc, 1, L), vL = pb(sc, 2, L), wL = NDIM == 3 ? pb(sc, 3, L) : 0.0, TL = pb(sc, 7, L);
                const double tra_n = GB[0 * NCOL + L] + dyu, tra_a = GB[1 * NCOL + L] + dyv;
                const double trb_n = NDIM == 3 ? GB[2 * NCOL + L] + dzu : 0.0, trb_b = NDIM == 3 ? GB[3 * NCOL + L] + dzw : 0.0;
                vx = ark_visc_face(KV, wc.u - uL, wc.v - vL, wc.w - wL, tra_n, tra_a, trb_n, trb_b,
                                   uL + wc.u, vL + wc.v, wL + wc.w, wc.T - TL);
                VB[0 * NCOL + tc] = vx.t0; VB[1 * NCOL + tc] = vx.t1; VB[3 * NCOL + tc] = vx.fe;
                if (NDIM == 3) VB[2 * NCOL + tc] = vx.t2;
            }
            if (do_update && inVy) {   // face (cj-1 | cj), normal y, transverse a = x, b = z
                const int L = tc - RX;
                const double uL = pb(sc, 1, L), vL = pb(sc, 2, L), wL = NDIM == 3 ? pb(sc, 3, L) : 0.0, TL = pb(sc, 7, L);
                const double tra_n = GB[4 * NCOL + L] + dxv, tra_a = GB[5 * NCOL + L] + dxu;
                const double trb_n = NDIM == 3 ? GB[6 * NCOL + L] + dzv : 0.0, trb_b = NDIM == 3 ? GB[3 * NCOL + L] + dzw : 0.0;
                vy = ark_visc_face(KV, wc.v - vL, wc.u - uL, wc.w - wL, tra_n, tra_a, trb_n, trb_b,
                                   vL + wc.v, uL + wc.u, wL + wc.w, wc.T - TL);
                // stored as (tau_yx, tau_yy, tau_yz, fe): component order x,y,z
                VB[4 * NCOL + tc] = vy.t1; VB[5 * NCOL + tc] = vy.t0; VB[7 * NCOL + tc] = vy.fe;
                if (NDIM == 3) VB[6 * NCOL + tc] = vy.t2;
            }
            if (NDIM == 3) {
                if (inU && q >= k0)    // face (q-1 | q), normal z, transverse a = x, b = y
                    vz = ark_visc_face(KV, wc.w - wmw, wc.u - wmu, wc.v - wmv, gpz[0] + dxw, gpz[1] + dxu, gpz[2] + dyw, gpz[3] + dyv,
                                       wmw + wc.w, wmu + wc.u, wmv + wc.v, wc.T - wmT);
                gpz[0] = dxw; gpz[1] = dxu; gpz[2] = dyw; gpz[3] = dyv;
            }
        }
        __syncthreads();                                       // (C) U~(q) and viscous fluxes visible

        // ---------------- S4: transport + update
        if (inU) {
            double Gz[5] = {0, 0, 0, 0, 0};       // full flux through the z face (q-1|q)
            double mzf = 0.0;
            if (NDIM == 3 && q >= k0) {
                const bool up = zlo.us >= 0.0;                  // PAPER.md:174, reading A10
                for (int f = 0; f < 5; ++f) Gz[f] = (up ? Utprev[f] : Ut[f]) * zlo.us;
                mzf = Gz[0];
                Gz[3] += zlo.pi;
                Gz[4] += zlo.pi * zlo.us;
                if (VISC) { Gz[1] -= vz.t1; Gz[2] -= vz.t2; Gz[3] -= vz.t0; Gz[4] -= vz.fe; }
                if (q > k0) {
                    // complete and store U^{n+1}(q-1):  acc - lam * G_z(high) + gravity work of the high face
                    double out[5];
                    for (int f = 0; f < 5; ++f) out[f] = acc[f] - lam * Gz[f];
                    if (ghz != 0.0) out[4] += dt * P.g[2] * (mzf < 0.0 ? mzf : 0.0);
                    double* __restrict__ c = Ocol + pstride * (long long)(q - 1);
                    c[0] = out[0];
                    c[fs] = out[1];
                    c[2 * fs] = out[2];
                    c[3 * fs] = out[3];
                    c[FE * fs] = out[4];
                    if (rate_scratch) rate_max = ark_umax(rate_max, ark_rate_epilogue(P, 3, out[0], out[1], out[2], out[3], out[4], inv_h, dcoef));
                }
            }
            if (do_update) {
                // in-plane faces of plane q: F = U~_up u* + (0, Pi* e_d, Pi* u*) - D ; dG = sum_d (F_d+ - F_d-)
                double dG[5];
                double work = 0.0;
                {   // x axis
                    const double usl = fx.us, ush = usxh;
                    const int nl = usl >= 0.0 ? tc - 1 : tc, nh = ush >= 0.0 ? tc : tc + 1;
                    const double ml = TB[nl] * usl, mh = TB[nh] * ush;
                    dG[0] = mh - ml;
                    dG[1] = (TB[NCOL + nh] * ush + pixh) - (TB[NCOL + nl] * usl + fx.pi);
                    dG[2] = TB[2 * NCOL + nh] * ush - TB[2 * NCOL + nl] * usl;
                    dG[3] = NDIM == 3 ? TB[3 * NCOL + nh] * ush - TB[3 * NCOL + nl] * usl : 0.0;
                    dG[4] = (TB[4 * NCOL + nh] + pixh) * ush - (TB[4 * NCOL + nl] + fx.pi) * usl;
                    if (gx_on) work += P.g[0] * ((ml > 0.0 ? ml : 0.0) + (mh < 0.0 ? mh : 0.0));
                }
                {   // y axis
                    const double usl = fy.us, ush = usyh;
                    const int nl = usl >= 0.0 ? tc - RX : tc, nh = ush >= 0.0 ? tc : tc + RX;
                    const double ml = TB[nl] * usl, mh = TB[nh] * ush;
                    dG[0] += mh - ml;
                    dG[1] += TB[NCOL + nh] * ush - TB[NCOL + nl] * usl;
                    dG[2] += (TB[2 * NCOL + nh] * ush + piyh) - (TB[2 * NCOL + nl] * usl + fy.pi);
                    if (NDIM == 3) dG[3] += TB[3 * NCOL + nh] * ush - TB[3 * NCOL + nl] * usl;
                    dG[4] += (TB[4 * NCOL + nh] + piyh) * ush - (TB[4 * NCOL + nl] + fy.pi) * usl;
                    if (gy_on) work += P.g[1] * ((ml > 0.0 ? ml : 0.0) + (mh < 0.0 ? mh : 0.0));
                }
                if (VISC) {
                    dG[1] -= (VB[0 * NCOL + tc + 1] - vx.t0) + (VB[4 * NCOL + tc + RX] - vy.t1);
                    dG[2] -= (VB[1 * NCOL + tc + 1] - vx.t1) + (VB[5 * NCOL + tc + RX] - vy.t0);
                    if (NDIM == 3) dG[3] -= (VB[2 * NCOL + tc + 1] - vx.t2) + (VB[6 * NCOL + tc + RX] - vy.t2);
                    dG[4] -= (VB[3 * NCOL + tc + 1] - vx.fe) + (VB[7 * NCOL + tc + RX] - vy.fe);
                }
                double nw[5];
                nw[0] = Ucur[0] - lam * dG[0];
                nw[1] = Ucur[1] - lam * dG[1] + lam * Six;
                nw[2] = Ucur[2] - lam * dG[2] + lam * Siy;
                nw[3] = Ucur[3] - lam * dG[3];
                nw[4] = Ucur[4] - lam * dG[4] + dt * work;
                if (NDIM == 3) {
                    // low z face enters with +lam*G_z and the gravity work dt g_z max(m,0); the source lam*S_i
                    for (int f = 0; f < 5; ++f) acc[f] = nw[f] + lam * Gz[f];
                    if (ghz != 0.0) {
                        acc[3] += lam * Siz;
                        acc[4] += dt * P.g[2] * (mzf > 0.0 ? mzf : 0.0);
                    }
                } else {
                    double* __restrict__ c = Ocol;
                    c[0] = nw[0];
                    c[fs] = nw[1];
                    c[2 * fs] = nw[2];
                    c[FE * fs] = nw[4];
                    if (rate_scratch) rate_max = ark_umax(rate_max, ark_rate_epilogue(P, 2, nw[0], nw[1], nw[2], 0.0, nw[4], inv_h, dcoef));
                }
            }
        }
        if (NDIM == 3) {
            // rotate the z pipeline
            for (int f = 0; f < 5; ++f) { Utprev[f] = Ut[f]; Ucur[f] = Unext[f]; Unext[f] = Upre[f]; }
            if (VISC) { wmu = wc.u; wmv = wc.v; wmw = wc.w; wmT = wc.T; }
            wc = wn;
            zlo = zhi;
            sc ^= 1; sn ^= 1;
        }
    }

    if (rate_scratch) {
        // block-wide max of the rate bit patterns -> one double per block
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
        if (t == 0) rate_scratch[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = ark_rate_from_bits(m);
    }
}
