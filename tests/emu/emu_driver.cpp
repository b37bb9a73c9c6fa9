// emu_driver.cpp -- TEST-ONLY: runs the CUDA kernel sources under the host emulation shim (ark_emu.h) so that the
// kernels' logic can be compared with the oracle without a GPU.  Mirrors the launch sequence of csrc/ark.cu
// (pack, ghost fill x/y/z, fused step, unpack; standalone CFL passes) with a small tile so that a tiny grid
// still spans several tiles, a ragged tail and several z chunks.
#define ARK_HOST_EMU 1
#define ARK_REG_RING 96
#define ARK_REG_TILE 208
#include "ark_emu.h"
#include "../../paper_1903_09043_b200/csrc/ark_step3d.cuh"

#include <cstring>

namespace {
constexpr int ETX = 8, ETY = 4;   // emulation tile
constexpr int ENW = 4;            // 3D: row pairs per block (region 12 x 8, tile 8 x 4) on ENW + 2 "warps" of 12 threads

ArkParams make_params(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
                      int theta, const int* bt, const double* bv) {
    ArkParams P;
    std::memset(&P, 0, sizeof P);
    P.nx = nx; P.ny = ny; P.nz = nz; P.ndim = nz > 1 ? 3 : 2; P.nf = nz > 1 ? 5 : 4;
    P.px = (nx + ARK_XOFF + ARK_NG + 15) / 16 * 16; P.py = ny + 4; P.pz = nz > 1 ? nz + 4 : 1; P.offz = nz > 1 ? 2 : 0;
    P.fstride = ((long long)P.px * P.py * P.pz + 31) / 32 * 32;
    P.h = h; P.gamma = gamma; P.gm1 = gamma - 1.0; P.mu = mu; P.kappa = kappa; P.theta = theta;
    for (int d = 0; d < 3; ++d) {
        P.g[d] = d < P.ndim ? g[d] : 0.0;
        for (int s = 0; s < 2; ++s) { P.bc[d][s] = bt[2 * d + s]; P.bcv[d][s] = bv[2 * d + s]; }
    }
    ark_fill_derived(P);
    return P;
}

template <int AXIS>
void bc(const ArkParams& P, double* U, long long n) {
    emu_dim3 g; g.x = (unsigned)((n + 63) / 64);
    ark_emu_launch(g, 64, 0, [&] { ark_k_bc<AXIS>(P, U); });
}

template <int NDIM, bool VISC>
void step(const ArkParams& P, const double* Uin, double* Uout, double dt, double* scratch, int zchunk, emu_dim3 grid) {
    const bool gen = P.phi != nullptr || P.eform != 0;        // mirrors do_step in csrc/ark.cu
    if constexpr (NDIM == 3) {
        using C = ArkCfg3<VISC, ETX, ENW>;
        static_assert(C::TY == ETY, "emulation tile");
        const bool gxy = P.D.g_on[0] || P.D.g_on[1];
        if (gen)      ark_emu_launch(grid, C::NT, C::SMEM_BYTES, [&] { ark_k_step3<VISC, true, true, ETX, ENW>(P, Uin, Uout, dt, nullptr, scratch, zchunk); }, C::RX);
        else if (gxy) ark_emu_launch(grid, C::NT, C::SMEM_BYTES, [&] { ark_k_step3<VISC, true, false, ETX, ENW>(P, Uin, Uout, dt, nullptr, scratch, zchunk); }, C::RX);
        else          ark_emu_launch(grid, C::NT, C::SMEM_BYTES, [&] { ark_k_step3<VISC, false, false, ETX, ENW>(P, Uin, Uout, dt, nullptr, scratch, zchunk); }, C::RX);
    } else {
        using C = ArkStepCfg<NDIM, VISC, ETX, ETY>;
        if (gen) ark_emu_launch(grid, C::NT, C::SMEM_BYTES, [&] { ark_k_step<NDIM, VISC, true, ETX, ETY>(P, Uin, Uout, dt, nullptr, scratch); });
        else     ark_emu_launch(grid, C::NT, C::SMEM_BYTES, [&] { ark_k_step<NDIM, VISC, false, ETX, ETY>(P, Uin, Uout, dt, nullptr, scratch); });
    }
}
}  // namespace

extern "C" {

// Advances the dense state by nsteps prescribed steps through the emulated kernels.  rates_out[s] receives the
// max CFL rate of the state AFTER step s as produced by the fused epilogue + pass 2; rate0_out the standalone
// two-pass reduction of the initial state.  zchunk <= 0 picks nz (one chunk).
int emu_run(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa, int theta,
            const int* bt, const double* bv, double* rho, double* rhou, double* rhov, double* rhow, double* E,
            int nsteps, const double* dts, int zchunk, double* rates_out, double* rate0_out, double* padded_out,
            int eform, const double* phi) {
    ArkParams P = make_params(nx, ny, nz, h, gamma, g, mu, kappa, theta, bt, bv);
    P.eform = eform;
    std::vector<double> A((size_t)P.nf * P.fstride, 0.0), B((size_t)P.nf * P.fstride, 0.0);
    std::vector<double> PhiPad;
    if (phi) {
        // mirrors ark_set_potential in csrc/ark.cu: pack, ghost sweeps x, y, z, all gravity terms on
        PhiPad.assign((size_t)P.fstride, 0.0);
        emu_dim3 gp; gp.x = (unsigned)(((long long)nx * ny * nz + 63) / 64);
        ark_emu_launch(gp, 64, 0, [&] { ark_k_pack(P, PhiPad.data(), phi, 0); });
        emu_dim3 g0; g0.x = (unsigned)(((long long)ny * nz + 63) / 64);
        ark_emu_launch(g0, 64, 0, [&] { ark_k_phi_ghosts<0>(P, PhiPad.data()); });
        emu_dim3 g1; g1.x = (unsigned)(((long long)(nx + 4) * nz + 63) / 64);
        ark_emu_launch(g1, 64, 0, [&] { ark_k_phi_ghosts<1>(P, PhiPad.data()); });
        if (P.ndim == 3) {
            emu_dim3 g2; g2.x = (unsigned)(((long long)(nx + 4) * (ny + 4) + 63) / 64);
            ark_emu_launch(g2, 64, 0, [&] { ark_k_phi_ghosts<2>(P, PhiPad.data()); });
        }
        P.phi = PhiPad.data();
        for (int d = 0; d < P.ndim; ++d) P.D.g_on[d] = 1;
    }
    std::vector<double> scratch(1 << 16, -1.0), result(8, 0.0);   // [0] max rate, [1] dt, [3] sticky non-finite flag
    double* dense[5] = {rho, rhou, rhov, P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)nx * ny * nz;
    emu_dim3 g1; g1.x = (unsigned)((n + 63) / 64);
    for (int f = 0; f < P.nf; ++f)
        ark_emu_launch(g1, 64, 0, [&] { ark_k_pack(P, A.data(), dense[f], f); });
    if (rate0_out) {
        emu_dim3 gg; gg.x = 3;
        ark_emu_launch(gg, 64, 0, [&] { ark_k_cfl_pass1(P, A.data(), scratch.data()); });
        emu_dim3 one;
        ark_emu_launch(one, 64, 0, [&] { ark_k_cfl_pass2(scratch.data(), 3, 1.0, result.data(), nullptr, nullptr); });
        *rate0_out = result[0];
    }
    double* cur = A.data();
    double* nxt = B.data();
    emu_dim3 grid;
    grid.x = (nx + ETX - 1) / ETX; grid.y = (ny + ETY - 1) / ETY;
    if (zchunk <= 0) zchunk = nz;
    grid.z = P.ndim == 3 ? (nz + zchunk - 1) / zchunk : 1;
    const bool visc = mu > 0.0 || kappa > 0.0;
    for (int s = 0; s < nsteps; ++s) {
        if (P.bc[0][0] == ARK_BCK_PERIODIC && s > 0) {
            // mirrors launch_bc in csrc/ark.cu: the step kernel wrote the periodic x ghost columns itself
        } else if (P.bc[0][0] == ARK_BCK_PERIODIC) {
            emu_dim3 gp; gp.x = (unsigned)((2LL * ny * nz * P.nf + 63) / 64);
            ark_emu_launch(gp, 64, 0, [&] { ark_k_bc_x_periodic(P, cur); });
        } else {
            bc<0>(P, cur, 2LL * ny * nz);
        }
        if (!(P.ndim == 2 && s > 0 && P.bc[0][0] == ARK_BCK_PERIODIC && P.bc[1][0] == ARK_BCK_PERIODIC))   // (2D, fully periodic: the step kernel wrote them)
            bc<1>(P, cur, 2LL * (nx + 4) * nz);
        if (P.ndim == 3) bc<2>(P, cur, 2LL * (nx + 4) * (ny + 4));
        if (s == 0 && padded_out) {
            const int mx = nx + 4;
            for (int f = 0; f < P.nf; ++f)
                for (long long r = 0; r < (long long)P.py * P.pz; ++r)
                    for (int i = 0; i < mx; ++i)
                        padded_out[(size_t)f * mx * P.py * P.pz + r * mx + i] = cur[f * P.fstride + r * P.px + i + (ARK_XOFF - ARK_NG)];
        }
        if (P.ndim == 3) { if (visc) step<3, true>(P, cur, nxt, dts[s], scratch.data(), zchunk, grid); else step<3, false>(P, cur, nxt, dts[s], scratch.data(), zchunk, grid); }
        else             { if (visc) step<2, true>(P, cur, nxt, dts[s], scratch.data(), zchunk, grid); else step<2, false>(P, cur, nxt, dts[s], scratch.data(), zchunk, grid); }
        std::swap(cur, nxt);
        if (rates_out) {
            emu_dim3 one;
            const int nv = (int)(grid.x * grid.y * grid.z);
            ark_emu_launch(one, 64, 0, [&] { ark_k_cfl_pass2(scratch.data(), nv, 1.0, result.data(), nullptr, nullptr); });
            rates_out[s] = result[0];
        }
    }
    for (int f = 0; f < P.nf; ++f)
        ark_emu_launch(g1, 64, 0, [&] { ark_k_unpack(P, cur, dense[f], f); });
    return 0;
}

}  // extern "C"
