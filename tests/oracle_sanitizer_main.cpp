// Stand-alone driver of the ORACLE for the sanitizer test (tests/test_oracle_pins.py::test_oracle_is_clean_under_asan_ubsan;
// SURVEY section 5): small 2D and 3D cases with every wall kind, all three energy forms, an array-valued potential, the
// ghost fill, the CFL rate and the diagnostics, built with -fsanitize=address,undefined.  Test infrastructure only; it
// calls the oracle's C entry points and checks nothing but return codes and finiteness (the pins check the values).
#include <cmath>
#include <cstdio>
#include <vector>

extern "C" {
int oracle_run_phi(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa, int theta,
                   const int* bc_type, const double* bc_val, double* rho, double* rhou, double* rhov, double* rhow, double* E,
                   int nsteps, double cfl, const double* dts, double* dts_out, int form, const double* phi);
double oracle_max_rate(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa, int theta,
                       const int* bc_type, const double* bc_val, const double* rho, const double* rhou, const double* rhov,
                       const double* rhow, const double* E);
int oracle_fill_ghosts(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa, int theta,
                       const int* bc_type, const double* bc_val, const double* rho, const double* rhou, const double* rhov,
                       const double* rhow, const double* E, double* prho, double* prhou, double* prhov, double* prhow, double* pE);
void oracle_diagnostics(int nx, int ny, int nz, double h, double gamma, const double* g, const double* rho, const double* rhou,
                        const double* rhov, const double* rhow, const double* E, double* out);
}

namespace {
unsigned long long lcg = 0x9E3779B97F4A7C15ull;
double unif() { lcg = lcg * 6364136223846793005ull + 1442695040888963407ull; return (double)(lcg >> 11) * (1.0 / 9007199254740992.0); }

int run_case(const char* name, int nx, int ny, int nz, const double g[3], double mu, double kappa, const int bct[6],
             const double bcv[6], int form, bool with_phi) {
    const size_t n = (size_t)nx * ny * nz;
    const double h = 1.0 / (nx > ny ? nx : ny), gamma = 1.4;
    std::vector<double> rho(n), mx(n), my(n), mz(n), E(n), phi(n);
    for (size_t c = 0; c < n; ++c) {
        const double r = 1.0 + 0.3 * (unif() - 0.5), p = 1.0 + 0.3 * (unif() - 0.5);
        const double u = 0.2 * (unif() - 0.5), v = 0.2 * (unif() - 0.5), w = nz > 1 ? 0.2 * (unif() - 0.5) : 0.0;
        rho[c] = r; mx[c] = r * u; my[c] = r * v; mz[c] = r * w;
        E[c] = p / (gamma - 1.0) + 0.5 * r * (u * u + v * v + w * w);
        const size_t i = c % nx, j = (c / nx) % ny, k = c / ((size_t)nx * ny);
        phi[c] = 0.8 * (j + 0.5) * h + 0.4 * (k + 0.5) * h * (k + 0.5) * h + 0.1 * std::sin(6.283185307179586 * (i + 0.5) / nx);
    }
    double* pw = nz > 1 ? mz.data() : nullptr;
    const size_t np = (size_t)(nx + 4) * (ny + 4) * (nz > 1 ? nz + 4 : 1);
    std::vector<double> P0(np), P1(np), P2(np), P3(np), P4(np);
    if (oracle_fill_ghosts(nx, ny, nz, h, gamma, g, mu, kappa, 1, bct, bcv, rho.data(), mx.data(), my.data(), pw, E.data(),
                           P0.data(), P1.data(), P2.data(), nz > 1 ? P3.data() : nullptr, P4.data()) != 0) return 1;
    const double rate = oracle_max_rate(nx, ny, nz, h, gamma, g, mu, kappa, 1, bct, bcv, rho.data(), mx.data(), my.data(), pw, E.data());
    if (!(rate > 0.0) || !std::isfinite(rate)) return 2;
    std::vector<double> dts(3);
    if (oracle_run_phi(nx, ny, nz, h, gamma, g, mu, kappa, 1, bct, bcv, rho.data(), mx.data(), my.data(), pw, E.data(), 3, 0.4,
                       nullptr, dts.data(), form, with_phi ? phi.data() : nullptr) != 0) return 3;
    double d[6];
    oracle_diagnostics(nx, ny, nz, h, gamma, g, rho.data(), mx.data(), my.data(), pw, E.data(), d);
    for (int q = 0; q < 6; ++q) if (!std::isfinite(d[q])) return 4;
    for (size_t c = 0; c < n; ++c) if (!std::isfinite(rho[c]) || !std::isfinite(E[c])) return 5;
    std::printf("%-28s ok  (dt %.3e, mass %.6f)\n", name, dts[2], d[4]);
    return 0;
}
}  // namespace

int main() {
    enum { PER = 0, REF = 1, FIX = 2, FLUX = 3 };
    int bad = 0;
    {   // 2D: periodic x, fixed-T bottom / reflecting top, gravity, viscous; normative form and eq. (11) form
        const double g[3] = {0.0, -1.0, 0.0};
        const int t[6] = {PER, PER, FIX, REF, PER, PER};
        const double v[6] = {0, 0, 2.5, 0, 0, 0};
        bad |= run_case("2d walls, form 0", 19, 13, 1, g, 2e-3, 3e-3, t, v, 0, false);
        bad |= run_case("2d walls, form 1", 19, 13, 1, g, 2e-3, 3e-3, t, v, 1, false);
    }
    {   // 3D: walls on every axis, oblique gravity, imposed-flux bottom wall
        const double g[3] = {0.2, -0.3, -1.0};
        const int t[6] = {REF, FIX, FIX, REF, FLUX, REF};
        const double v[6] = {0, 2.5, 3.5, 0, 0.03, 0};
        bad |= run_case("3d all walls + flux wall", 11, 9, 10, g, 1e-3, 5e-2, t, v, 0, false);
    }
    {   // 3D: array-valued potential, Appendix-B energy form, walls in y and z
        const double g[3] = {0.0, 0.0, 0.0};
        const int t[6] = {PER, PER, REF, REF, FIX, REF};
        const double v[6] = {0, 0, 0, 0, 2.5, 0};
        bad |= run_case("3d phi + appendix B", 10, 8, 9, g, 1e-3, 2e-3, t, v, 2, true);
    }
    {   // 3D: fully periodic, inviscid
        const double g[3] = {0.0, 0.0, 0.0};
        const int t[6] = {PER, PER, PER, PER, PER, PER};
        const double v[6] = {0, 0, 0, 0, 0, 0};
        bad |= run_case("3d periodic inviscid", 8, 7, 6, g, 0.0, 0.0, t, v, 0, false);
    }
    return bad;
}
