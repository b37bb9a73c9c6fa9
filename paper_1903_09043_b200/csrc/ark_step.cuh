// ark_step.cuh -- the fused full-step kernel (acoustic + transport + dissipative + update + CFL epilogue).
//
// One launch advances U^n -> U^{n+1}: every conserved field is read once and written once
// (80 B per cell update in 3D, 64 B in 2D), all face quantities and the intermediate state U~
// live in registers / shared memory only.
//
// Decomposition ("2.5-D marching"): a block owns a TX x TY tile of (x,y) columns plus a 2-cell halo
// (region RX x RY, one thread per column, threads linearised over the region so that consecutive
// lanes touch consecutive shared-memory words) and marches along z over a chunk of planes.
// Per plane q one iteration does
//   S1  primitives of plane q+1 (own column)                       -> smem ring PB (3 planes)
//   S2  acoustic faces x-,y- of plane q (neighbours from PB), z face (q|q+1) from registers,
//       viscous/heat fluxes of the x-,y- faces of plane q          -> smem FB, VB
//   S3  acoustic update U~(q) on tile + 1 ring   -> smem TB (2 planes)
//   S4  transport fluxes (upwind on u*) of the in-plane faces of plane q and of the
//       z face (q-1|q); completes and stores U^{n+1}(q-1); folds the CFL rate of the new state
//       into a per-block maximum.
// z neighbours of a column stay in the owning thread's registers; only x/y neighbours go through
// shared memory.
#pragma once
#include "ark_device.cuh"

#define ARK_NPRIM 8   // rho,u,v,w,p,rc,irc,T

template <int TX, int TY>
struct ArkStepCfg {
    static constexpr int RX = TX + 4, RY = TY + 4, NCOL = RX * RY;
    static constexpr int NT = ((NCOL + 31) / 32) * 32;
    // shared memory (doubles): PB[3][NPRIM][NCOL] FB[6][NCOL] VB[8][NCOL] TB[2][5][NCOL] red[32]
    static constexpr int SMEM_DOUBLES = (3 * ARK_NPRIM + 6 + 8 + 10) * NCOL + 32;
    static constexpr size_t SMEM_BYTES = (size_t)SMEM_DOUBLES * sizeof(double);
};

// transverse-gradient part of a viscous face flux; see ark_visc_face below
struct ArkVisc { double t0, t1, t2, fe; };

// Dissipative flux through a face with unit normal along axis d (tau = mu(grad u + grad u^T)
// + eta div u I, eta = -2/3 mu; divergence form, Fourier flux; stencil = reading A6).
//   dn[3]   : (u,v,w)_R - (u,v,w)_L                       (normal differences, un-normalised)
//   tr_a[2] : sum over the two adjacent cells of the centred difference along transverse axis a of
//             (u_d, u_a)  -> d_a u_d and d_a u_a at the face are tr/(4h)
//   tr_b[2] : same for transverse axis b
//   ub[3]   : (u,v,w)_L + (u,v,w)_R                       (2 x face velocity)
//   dT      : T_R - T_L
// Returns tau_{d,.} ordered (normal, a, b) and the energy flux tau.ubar + kappa dT/h.
ARK_DEV ArkVisc ark_visc_face(const ArkParams& P, double inv_h, double dn_n, double dn_a, double dn_b,
                              double tra_n, double tra_a, double trb_n, double trb_b,
                              double ub_n, double ub_a, double ub_b, double dT) {
    ArkVisc r;
    const double q = 0.25 * inv_h;
    const double gnn = dn_n * inv_h;                  // d_d u_d
    const double gaa = tra_a * q;                     // d_a u_a
    const double gbb = trb_b * q;                     // d_b u_b
    const double div = gnn + gaa + gbb;
    r.t0 = P.mu * (2.0 * gnn) - (2.0 / 3.0) * P.mu * div;
    r.t1 = P.mu * (dn_a * inv_h + tra_n * q);         // mu (d_d u_a + d_a u_d)
    r.t2 = P.mu * (dn_b * inv_h + trb_n * q);
    r.fe = 0.5 * (r.t0 * ub_n + r.t1 * ub_a + r.t2 * ub_b) + P.kappa * (dT * inv_h);
    return r;
}

template <int NDIM, bool VISC, int TX, int TY>
ARK_GLOBAL void
#ifndef ARK_HOST_EMU
__launch_bounds__(ArkStepCfg<TX, TY>::NT, 1)
#endif
ark_k_step(const ArkParams P, const double* __restrict__ Uin, double* __restrict__ Uout,
           double dt_value, const double* __restrict__ dt_dev, double* __restrict__ rate_scratch, int zchunk) {
    using C = ArkStepCfg<TX, TY>;
    constexpr int RX = C::RX, NCOL = C::NCOL;
    constexpr int NF = NDIM == 3 ? 5 : 4;
    constexpr int FE = NF - 1;                        // index of the energy field in HBM
    ARK_DYN_SMEM(smem);
    double* PB = smem;                                // [3][NPRIM][NCOL]
    double* FB = PB + 3 * ARK_NPRIM * NCOL;           // [6][NCOL]: usx,pix,usy,piy,Sx,Sy (low faces of plane q)
    double* VB = FB + 6 * NCOL;                       // [8][NCOL]: viscous low-face fluxes x(4), y(4)
    double* TB = VB + 8 * NCOL;                       // [2][5][NCOL]: U~ planes
    double* red = TB + 10 * NCOL;                     // [32]

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

    // roles
    const bool inA = live && ci >= 1 && ci <= RX - 2 && cj >= 1 && cj <= C::RY - 2 && gi <= P.nx && gj <= P.ny;
    const bool inFx = live && ci >= 1 && cj >= 1 && cj <= C::RY - 2;      // owns the low-x face (ci-1 | ci)
    const bool inFy = live && cj >= 1 && ci >= 1 && ci <= RX - 2;         // owns the low-y face (cj-1 | cj)
    const bool inU = live && ci >= 2 && ci < 2 + TX && cj >= 2 && cj < 2 + TY && gi < P.nx && gj < P.ny;
    const bool inVx = VISC && live && ci >= 2 && ci <= 2 + TX && cj >= 2 && cj < 2 + TY;
    const bool inVy = VISC && live && cj >= 2 && cj <= 2 + TY && ci >= 2 && ci < 2 + TX;

    const double dt = dt_dev ? dt_dev[1] : dt_value;
    const double inv_h = 1.0 / P.h;
    const double lam = dt * inv_h;
    const double ghx = P.g[0] * P.h, ghy = P.g[1] * P.h, ghz = P.g[2] * P.h;
    const int th = P.theta;
    const double dcoef = 2.0 * P.ndim * fmax(4.0 * P.mu / 3.0, P.gm1 * P.kappa) * inv_h * inv_h;

    const long long colbase = (long long)(li + ARK_NG) + (long long)P.px * (long long)(lj + ARK_NG);
    const long long pstride = (long long)P.px * P.py;
    auto gidx = [&](int k) -> long long { return colbase + pstride * (long long)(k + P.offz); };

    auto loadU = [&](int k, double* u5) {
        const long long c = gidx(k);
        u5[0] = Uin[c];
        u5[1] = Uin[P.fstride + c];
        u5[2] = Uin[2 * P.fstride + c];
        u5[3] = NDIM == 3 ? Uin[3 * P.fstride + c] : 0.0;
        u5[4] = Uin[FE * P.fstride + c];
    };
    auto pb = [&](int slot, int f, int col) -> double& { return PB[(slot * ARK_NPRIM + f) * NCOL + col]; };
    auto storePrim = [&](int slot, const ArkPrim& w) {
        pb(slot, 0, tc) = w.rho; pb(slot, 1, tc) = w.u; pb(slot, 2, tc) = w.v; pb(slot, 3, tc) = w.w;
        pb(slot, 4, tc) = w.p; pb(slot, 5, tc) = w.rc; pb(slot, 6, tc) = w.irc; pb(slot, 7, tc) = w.T;
    };

    double rate_max = -1.0;

    // ---------------------------------------------------------------------------------------------
    // register pipeline along z
    // ---------------------------------------------------------------------------------------------
    double Ucur[5], Unext[5];          // U^n(q), U^n(q+1)
    ArkPrim wm, wc, wn;                // primitives of own column at q-1, q, q+1
    ArkFace zlo = {0, 0, 0}, zhi = {0, 0, 0};   // acoustic z faces (q-1|q), (q|q+1)
    double Utprev[5] = {0, 0, 0, 0, 0};         // U~(q-1) of own column
    double acc[5] = {0, 0, 0, 0, 0};            // U^{n+1}(q-1) minus its high-z flux
    int sm = 0, sc = 1, sn = 2;        // PB slots of planes q-1, q, q+1

    if (NDIM == 3) {
        // prologue: planes k0-2 and k0-1
        double Ua[5];
        loadU(k0 - 2, Ua);
        wm = ark_prim(P, Ua[0], Ua[1], Ua[2], Ua[3], Ua[4]);
        loadU(k0 - 1, Ucur);
        wc = ark_prim(P, Ucur[0], Ucur[1], Ucur[2], Ucur[3], Ucur[4]);
        storePrim(sm, wm);
        storePrim(sc, wc);
        zlo = ark_face(th, ghz, wm.rho, wm.w, wm.p, wm.rc, wm.irc, wc.rho, wc.w, wc.p, wc.rc, wc.irc);
        loadU(k0, Unext);
    } else {
        loadU(0, Unext);
        wm = wc = ark_prim(P, Unext[0], Unext[1], Unext[2], Unext[3], Unext[4]);
    }

    const int qbeg = NDIM == 3 ? k0 - 1 : 0, qend = NDIM == 3 ? k1 : 0;
    for (int q = qbeg; q <= qend; ++q) {
        // ---------------- S1: primitives of plane q+1 (3D) / plane 0 (2D)
        double Upre[5] = {0, 0, 0, 0, 0};
        if (NDIM == 3) {
            wn = ark_prim(P, Unext[0], Unext[1], Unext[2], Unext[3], Unext[4]);
            storePrim(sn, wn);
            if (q + 2 <= k1 + 1) loadU(q + 2, Upre);           // prefetch, consumed next iteration
        } else {
            for (int f = 0; f < 5; ++f) Ucur[f] = Unext[f];
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
            if (ghx != 0.0) FB[4 * NCOL + tc] = fx.S;
        }
        if (inFy) {
            const int n = tc - RX;
            fy = ark_face(th, ghy, pb(sc, 0, n), pb(sc, 2, n), pb(sc, 4, n), pb(sc, 5, n), pb(sc, 6, n),
                          wc.rho, wc.v, wc.p, wc.rc, wc.irc);
            FB[2 * NCOL + tc] = fy.us; FB[3 * NCOL + tc] = fy.pi;
            if (ghy != 0.0) FB[5 * NCOL + tc] = fy.S;
        }
        if (NDIM == 3)
            zhi = ark_face(th, ghz, wc.rho, wc.w, wc.p, wc.rc, wc.irc, wn.rho, wn.w, wn.p, wn.rc, wn.irc);

        // viscous / heat fluxes through the low x and low y faces of plane q
        ArkVisc vx = {0, 0, 0, 0}, vy = {0, 0, 0, 0};
        if (VISC && do_update) {
            if (inVx) {   // face (ci-1 | ci), normal x, transverse a = y, b = z
                const int L = tc - 1;
                const double uL = pb(sc, 1, L), vL = pb(sc, 2, L), wL = pb(sc, 3, L), TL = pb(sc, 7, L);
                const double tra_n = (pb(sc, 1, L + RX) - pb(sc, 1, L - RX)) + (pb(sc, 1, tc + RX) - pb(sc, 1, tc - RX));  // d_y u
                const double tra_a = (pb(sc, 2, L + RX) - pb(sc, 2, L - RX)) + (pb(sc, 2, tc + RX) - pb(sc, 2, tc - RX));  // d_y v
                double trb_n = 0.0, trb_b = 0.0;
                if (NDIM == 3) {
                    trb_n = (pb(sn, 1, L) - pb(sm, 1, L)) + (wn.u - wm.u);                                                  // d_z u
                    trb_b = (pb(sn, 3, L) - pb(sm, 3, L)) + (wn.w - wm.w);                                                  // d_z w
                }
                vx = ark_visc_face(P, inv_h, wc.u - uL, wc.v - vL, wc.w - wL, tra_n, tra_a, trb_n, trb_b,
                                   uL + wc.u, vL + wc.v, wL + wc.w, wc.T - TL);
                VB[0 * NCOL + tc] = vx.t0; VB[1 * NCOL + tc] = vx.t1; VB[2 * NCOL + tc] = vx.t2; VB[3 * NCOL + tc] = vx.fe;
            }
            if (inVy) {   // face (cj-1 | cj), normal y, transverse a = x, b = z
                const int L = tc - RX;
                const double uL = pb(sc, 1, L), vL = pb(sc, 2, L), wL = pb(sc, 3, L), TL = pb(sc, 7, L);
                const double tra_n = (pb(sc, 2, L + 1) - pb(sc, 2, L - 1)) + (pb(sc, 2, tc + 1) - pb(sc, 2, tc - 1));      // d_x v
                const double tra_a = (pb(sc, 1, L + 1) - pb(sc, 1, L - 1)) + (pb(sc, 1, tc + 1) - pb(sc, 1, tc - 1));      // d_x u
                double trb_n = 0.0, trb_b = 0.0;
                if (NDIM == 3) {
                    trb_n = (pb(sn, 2, L) - pb(sm, 2, L)) + (wn.v - wm.v);                                                  // d_z v
                    trb_b = (pb(sn, 3, L) - pb(sm, 3, L)) + (wn.w - wm.w);                                                  // d_z w
                }
                vy = ark_visc_face(P, inv_h, wc.v - vL, wc.u - uL, wc.w - wL, tra_n, tra_a, trb_n, trb_b,
                                   vL + wc.v, uL + wc.u, wL + wc.w, wc.T - TL);
                // stored as (tau_yx, tau_yy, tau_yz, fe): component order x,y,z
                VB[4 * NCOL + tc] = vy.t1; VB[5 * NCOL + tc] = vy.t0; VB[6 * NCOL + tc] = vy.t2; VB[7 * NCOL + tc] = vy.fe;
            }
        }
        // viscous / heat flux through the z face (q-1 | q): normal z, transverse a = x, b = y.  Computed here
        // (not in S4) because slot sm of PB is overwritten by S1 of the next iteration.
        ArkVisc vz = {0, 0, 0, 0};
        if (VISC && NDIM == 3 && inU && q >= k0) {
            const double tra_n = (pb(sm, 3, tc + 1) - pb(sm, 3, tc - 1)) + (pb(sc, 3, tc + 1) - pb(sc, 3, tc - 1));      // d_x w
            const double tra_a = (pb(sm, 1, tc + 1) - pb(sm, 1, tc - 1)) + (pb(sc, 1, tc + 1) - pb(sc, 1, tc - 1));      // d_x u
            const double trb_n = (pb(sm, 3, tc + RX) - pb(sm, 3, tc - RX)) + (pb(sc, 3, tc + RX) - pb(sc, 3, tc - RX));  // d_y w
            const double trb_b = (pb(sm, 2, tc + RX) - pb(sm, 2, tc - RX)) + (pb(sc, 2, tc + RX) - pb(sc, 2, tc - RX));  // d_y v
            vz = ark_visc_face(P, inv_h, wc.w - wm.w, wc.u - wm.u, wc.v - wm.v, tra_n, tra_a, trb_n, trb_b,
                               wm.w + wc.w, wm.u + wc.u, wm.v + wc.v, wc.T - wm.T);
        }
        __syncthreads();                                       // (B) faces visible

        // ---------------- S3: acoustic update U~(q), PAPER.md:158-160 (+ reading A3 for the energy)
        double Ut[5] = {0, 0, 0, 0, 0};
        double usxh = 0, pixh = 0, usyh = 0, piyh = 0, Six = 0, Siy = 0, Siz = 0;
        if (inA) {
            usxh = FB[0 * NCOL + tc + 1]; pixh = FB[1 * NCOL + tc + 1];
            usyh = FB[2 * NCOL + tc + RX]; piyh = FB[3 * NCOL + tc + RX];
            if (ghx != 0.0) Six = 0.5 * (fx.S + FB[4 * NCOL + tc + 1]);
            if (ghy != 0.0) Siy = 0.5 * (fy.S + FB[5 * NCOL + tc + RX]);
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
            double* tb = TB + (q & 1) * 5 * NCOL;
            tb[0 * NCOL + tc] = Ut[0]; tb[1 * NCOL + tc] = Ut[1]; tb[2 * NCOL + tc] = Ut[2];
            if (NDIM == 3) tb[3 * NCOL + tc] = Ut[3];
            tb[4 * NCOL + tc] = Ut[4];
        }
        __syncthreads();                                       // (C) U~(q) visible

        // ---------------- S4: transport + update
        if (inU) {
            const double* tb = TB + (q & 1) * 5 * NCOL;
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
                    out[4] += dt * P.g[2] * fmin(mzf, 0.0);
                    const long long c = gidx(q - 1);
                    Uout[c] = out[0];
                    Uout[P.fstride + c] = out[1];
                    Uout[2 * P.fstride + c] = out[2];
                    Uout[3 * P.fstride + c] = out[3];
                    Uout[FE * P.fstride + c] = out[4];
                    if (rate_scratch) rate_max = ark_nanmax(rate_max, ark_rate(P, out[0], out[1], out[2], out[3], out[4], inv_h, dcoef));
                }
            }
            if (do_update) {
                // in-plane faces of plane q: G = U~_up u* + (0, Pi* e_d, Pi* u*) - D
                double dG[5] = {0, 0, 0, 0, 0};
                double work = 0.0;
                {   // low x
                    const double us = fx.us;
                    const int n = us >= 0.0 ? tc - 1 : tc;
                    const double m = tb[n] * us;
                    dG[0] -= m; dG[1] -= tb[NCOL + n] * us + fx.pi; dG[2] -= tb[2 * NCOL + n] * us;
                    if (NDIM == 3) dG[3] -= tb[3 * NCOL + n] * us;
                    dG[4] -= (tb[4 * NCOL + n] + fx.pi) * us;
                    work += P.g[0] * fmax(m, 0.0);
                }
                {   // high x
                    const double us = usxh;
                    const int n = us >= 0.0 ? tc : tc + 1;
                    const double m = tb[n] * us;
                    dG[0] += m; dG[1] += tb[NCOL + n] * us + pixh; dG[2] += tb[2 * NCOL + n] * us;
                    if (NDIM == 3) dG[3] += tb[3 * NCOL + n] * us;
                    dG[4] += (tb[4 * NCOL + n] + pixh) * us;
                    work += P.g[0] * fmin(m, 0.0);
                }
                {   // low y
                    const double us = fy.us;
                    const int n = us >= 0.0 ? tc - RX : tc;
                    const double m = tb[n] * us;
                    dG[0] -= m; dG[1] -= tb[NCOL + n] * us; dG[2] -= tb[2 * NCOL + n] * us + fy.pi;
                    if (NDIM == 3) dG[3] -= tb[3 * NCOL + n] * us;
                    dG[4] -= (tb[4 * NCOL + n] + fy.pi) * us;
                    work += P.g[1] * fmax(m, 0.0);
                }
                {   // high y
                    const double us = usyh;
                    const int n = us >= 0.0 ? tc : tc + RX;
                    const double m = tb[n] * us;
                    dG[0] += m; dG[1] += tb[NCOL + n] * us; dG[2] += tb[2 * NCOL + n] * us + piyh;
                    if (NDIM == 3) dG[3] += tb[3 * NCOL + n] * us;
                    dG[4] += (tb[4 * NCOL + n] + piyh) * us;
                    work += P.g[1] * fmin(m, 0.0);
                }
                if (VISC) {
                    dG[1] -= VB[0 * NCOL + tc + 1] - vx.t0; dG[2] -= VB[1 * NCOL + tc + 1] - vx.t1;
                    if (NDIM == 3) dG[3] -= VB[2 * NCOL + tc + 1] - vx.t2;
                    dG[4] -= VB[3 * NCOL + tc + 1] - vx.fe;
                    dG[1] -= VB[4 * NCOL + tc + RX] - vy.t1; dG[2] -= VB[5 * NCOL + tc + RX] - vy.t0;
                    if (NDIM == 3) dG[3] -= VB[6 * NCOL + tc + RX] - vy.t2;
                    dG[4] -= VB[7 * NCOL + tc + RX] - vy.fe;
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
                    acc[3] += lam * Siz;
                    acc[4] += dt * P.g[2] * fmax(mzf, 0.0);
                } else {
                    const long long c = gidx(0);
                    Uout[c] = nw[0];
                    Uout[P.fstride + c] = nw[1];
                    Uout[2 * P.fstride + c] = nw[2];
                    Uout[FE * P.fstride + c] = nw[4];
                    if (rate_scratch) rate_max = ark_nanmax(rate_max, ark_rate(P, nw[0], nw[1], nw[2], 0.0, nw[4], inv_h, dcoef));
                }
            }
        }
        if (NDIM == 3) {
            // rotate the z pipeline
            for (int f = 0; f < 5; ++f) { Utprev[f] = Ut[f]; Ucur[f] = Unext[f]; Unext[f] = Upre[f]; }
            wm = wc; wc = wn;
            zlo = zhi;
            const int s = sm; sm = sc; sc = sn; sn = s;
        }
    }

    if (rate_scratch) {
        const double m = ark_block_nanmax(rate_max, red);
        if (t == 0) rate_scratch[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = m;
    }
}
