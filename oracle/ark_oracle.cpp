// ark_oracle.cpp -- ORACLE (test infrastructure, NOT the product).
//
// Plain, slow, single-threaded fp64 CPU implementation of one explicit time
// step of the all-Mach, well-balanced finite-volume scheme of
// Padioleau, Tremblin, Audit, Kestener & Kokh (arXiv 1903.09043), written
// directly from /root/reference/PAPER.md ("PAPER.md:<line>" below) with the
// readings A1..A26 listed in DESIGN.md.  It shares no code with the CUDA path
// under paper_1903_09043_b200/csrc/ and is only ever called from tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
//
// Build:  g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC   (oracle/build.py)
// No blocking, fusion or reordering beyond what the paper's algorithm states:
// the step is the literal sequence
//   1. ghost fill            (readings A9, A22)
//   2. primitives
//   3. acoustic face values
//   4. acoustic update -> U~ (reading A3)
//   5. transport (upwind on u*) + dissipative fluxes + conservative update
//
//   6. CFL time step         (reading A4)
// every intermediate being a full array so a reader can check each loop
// against the paper by eye.
//
// Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): P1 constant state
// bit-exact, P2 conservation of mass / transverse momentum / E+rho*Phi,
// P3 hydrostatic state (14) at rest + Table 1 magnitudes, P4 E-form ==
// calligraphic-E form (11), P5 g=0 reduction, P6 Sod vs exact Riemann
// solution, P7 Gresho kinetic-energy retention, P8 hand-computed face,
// P9 discrete Laplacian closed forms for the dissipative operator,
// P10 axis-permutation / mirror symmetry.  Parity unpinned: none of the
// functions below; Rayleigh-Benard onset curves / spectra (figures only) are
// not reproduced and are out of scope.

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>

namespace {

constexpr int NG = 2;          // ghost layers per side (reading A9)
constexpr double K_IMP = 1.1;  // a = K*max(rho_L c_L, rho_R c_R)  (reading A2)

enum { BC_PERIODIC = 0, BC_REFLECTING = 1, BC_FIXED_T = 2, BC_FLUX = 3 };

struct Cfg {
    int n[3];        // interior cells per axis; n[2]==1 -> 2D (reading A18)
    int ndim;        // 2 or 3
    double h;        // uniform cell size
    double gamma;    // ideal gas
    double g[3];     // constant gravity vector, Phi = -g.x (reading A12)
    double mu;       // dynamic viscosity
    double kappa;    // thermal conductivity
    int theta;       // 0: theta == 1 ; 1: eq. (13)
    int bc[3][2];    // [axis][lo,hi]
    double bcv[3][2];// wall temperature for BC_FIXED_T; heat flux entering the domain for BC_FLUX
    const double* phi; // optional gravitational potential at the interior cell centres (dense, x fastest; PAPER.md:55 general
                     // Phi(x)); NULL: Phi = -g.x with the constant vector g (reading A12).  Not owned.
};

struct Grid {
    int n[3], m[3], off[3];
    size_t ncell;
    explicit Grid(const Cfg& c) {
        for (int d = 0; d < 3; ++d) {
            n[d] = c.n[d];
            off[d] = (d < c.ndim) ? NG : 0;
            m[d] = n[d] + 2 * off[d];
        }
        ncell = (size_t)m[0] * m[1] * m[2];
    }
    // (i,j,k) are interior-based indices; ghosts are -2,-1 and n,n+1.
    size_t at(int i, int j, int k) const {
        return (size_t)(i + off[0]) + (size_t)m[0] * ((size_t)(j + off[1]) + (size_t)m[1] * (size_t)(k + off[2]));
    }
    size_t at(const int c[3]) const { return at(c[0], c[1], c[2]); }
    size_t stride(int d) const { return d == 0 ? 1 : (d == 1 ? (size_t)m[0] : (size_t)m[0] * m[1]); }
};

// q[0]=rho, q[1..3]=rho*u_d, q[4]=rho*E  (rho E = rho e + 1/2 rho u^2)
struct State {
    std::vector<double> q[5];
    explicit State(size_t n) { for (auto& v : q) v.assign(n, 0.0); }
};

struct Prim {
    std::vector<double> rho, u[3], p, c, T;
    explicit Prim(size_t n) : rho(n), p(n), c(n), T(n) { for (auto& v : u) v.assign(n, 0.0); }
};

// ---------------------------------------------------------------------------
// 2. primitives, one cell (PAPER.md:315-319 EOS and sound speed; :370 p = rho T)
// ---------------------------------------------------------------------------
struct CellPrim { double rho, u[3], p, c, T; };

CellPrim cons_to_prim(double gamma, double rho, double mx, double my, double mz, double E) {
    CellPrim w;
    const double rinv = 1.0 / rho;
    w.rho = rho;
    w.u[0] = mx * rinv;
    w.u[1] = my * rinv;
    w.u[2] = mz * rinv;
    const double ke = 0.5 * (mx * w.u[0] + my * w.u[1] + mz * w.u[2]);
    w.p = (gamma - 1.0) * (E - ke);
    w.c = std::sqrt(gamma * w.p * rinv);
    w.T = w.p * rinv;
    return w;
}

// ---------------------------------------------------------------------------
// 3. acoustic face values between cells L and R along one axis.
//    un = velocity component normal to the face, gh = g_d * h.
//    PAPER.md:152 (u*, Pi*, a, S), PAPER.md:218-222 (theta, eq. 13).
// ---------------------------------------------------------------------------
struct Face { double a, S, ustar, theta, pistar; };

Face acoustic_face(double rhoL, double unL, double pL, double cL,
                   double rhoR, double unR, double pR, double cR,
                   double gh, int theta_flag) {
    Face f;
    f.a = K_IMP * std::max(rhoL * cL, rhoR * cR);
    // S_{i+1/2} = -1/2 (rho_i + rho_{i+1}) (Phi_{i+1} - Phi_i),  Phi_{i+1}-Phi_i = -g_d h
    f.S = 0.5 * (rhoL + rhoR) * gh;
    f.ustar = 0.5 * (unL + unR) - (pR - pL - f.S) / (2.0 * f.a);
    if (theta_flag) {
        const double Ma = std::fabs(f.ustar) / std::max(cL, cR);
        f.theta = std::min(Ma, 1.0);
    } else {
        f.theta = 1.0;
    }
    f.pistar = 0.5 * (pL + pR) - 0.5 * f.a * f.theta * (unR - unL);
    return f;
}

// ---------------------------------------------------------------------------
// 1. ghost fill (reading A9).  Axis order x, y, z; each later axis sweeps the
//    already-extended range of the earlier ones so edges and corners are set.
// ---------------------------------------------------------------------------
// Padded potential for a run with an array-valued Phi (PAPER.md:55, :152 'Phi_{i+1} - Phi_i'): interior values from
// cfg.phi; ghost values (reading A25): periodic axes wrap, wall axes continue Phi linearly from the two cells next to
// the wall (Phi(-l) = Phi(0) + l (Phi(0) - Phi(1))), which reproduces a constant gravity exactly.  Same x, y, z sweep
// order over already-extended ranges as the state's ghost fill.  Empty when cfg.phi == NULL (constant g).
std::vector<double> padded_potential(const Cfg& cfg, const Grid& G) {
    std::vector<double> P;
    if (!cfg.phi) return P;
    P.assign(G.ncell, 0.0);
    size_t s = 0;
    for (int k = 0; k < G.n[2]; ++k) for (int j = 0; j < G.n[1]; ++j) for (int i = 0; i < G.n[0]; ++i, ++s) P[G.at(i, j, k)] = cfg.phi[s];
    for (int d = 0; d < cfg.ndim; ++d) {
        int lo[3], hi[3];
        for (int e = 0; e < 3; ++e) {
            if (e < d && e < cfg.ndim) { lo[e] = -NG; hi[e] = G.n[e] + NG; }
            else                       { lo[e] = 0;   hi[e] = G.n[e]; }
        }
        lo[d] = 0; hi[d] = 1;
        const int n = G.n[d];
        int c[3];
        for (c[2] = lo[2]; c[2] < hi[2]; ++c[2])
        for (c[1] = lo[1]; c[1] < hi[1]; ++c[1])
        for (c[0] = lo[0]; c[0] < hi[0]; ++c[0]) {
            auto at = [&](int i) { int q[3] = {c[0], c[1], c[2]}; q[d] = i; return G.at(q); };
            for (int l = 1; l <= NG; ++l) {
                if (cfg.bc[d][0] == BC_PERIODIC) {
                    P[at(-l)] = P[at(n - l)];
                    P[at(n - 1 + l)] = P[at(l - 1)];
                } else {
                    P[at(-l)] = P[at(0)] + l * (P[at(0)] - P[at(1)]);
                    P[at(n - 1 + l)] = P[at(n - 1)] + l * (P[at(n - 1)] - P[at(n - 2)]);
                }
            }
        }
    }
    return P;
}

void fill_ghosts(const Cfg& cfg, const Grid& G, State& U, const std::vector<double>& PhiP) {
    for (int d = 0; d < cfg.ndim; ++d) {
        int lo[3], hi[3];
        for (int e = 0; e < 3; ++e) {
            if (e < d && e < cfg.ndim) { lo[e] = -NG; hi[e] = G.n[e] + NG; }   // already extended
            else                       { lo[e] = 0;   hi[e] = G.n[e]; }
        }
        lo[d] = 0; hi[d] = 1;                                                  // the swept axis itself
        const int n = G.n[d];
        for (int side = 0; side < 2; ++side) {
            const int type = cfg.bc[d][side];
            for (int l = 1; l <= NG; ++l) {
                const int ig = side == 0 ? -l : n - 1 + l;          // ghost index along d
                int c[3];
                for (c[2] = lo[2]; c[2] < hi[2]; ++c[2])
                for (c[1] = lo[1]; c[1] < hi[1]; ++c[1])
                for (c[0] = lo[0]; c[0] < hi[0]; ++c[0]) {
                    int cg[3] = {c[0], c[1], c[2]}; cg[d] = ig;
                    const size_t jg = G.at(cg);
                    if (type == BC_PERIODIC) {
                        int cs[3] = {c[0], c[1], c[2]};
                        cs[d] = side == 0 ? n - l : l - 1;          // -1 <- n-1, -2 <- n-2 ; n <- 0, n+1 <- 1
                        const size_t js = G.at(cs);
                        for (int f = 0; f < 5; ++f) U.q[f][jg] = U.q[f][js];
                        continue;
                    }
                    // walls: mirror cell and previous cell of the hydrostatic chain (14)
                    int cs[3] = {c[0], c[1], c[2]}; cs[d] = side == 0 ? l - 1 : n - l;
                    int cp[3] = {c[0], c[1], c[2]}; cp[d] = side == 0 ? ig + 1 : ig - 1;
                    const size_t js = G.at(cs), jp = G.at(cp);
                    const CellPrim ws = cons_to_prim(cfg.gamma, U.q[0][js], U.q[1][js], U.q[2][js], U.q[3][js], U.q[4][js]);
                    const CellPrim wp = cons_to_prim(cfg.gamma, U.q[0][jp], U.q[1][jp], U.q[2][jp], U.q[3][jp], U.q[4][jp]);
                    double ug[3], Tg;
                    if (type == BC_REFLECTING) {
                        for (int e = 0; e < 3; ++e) ug[e] = (e == d) ? -ws.u[e] : ws.u[e];
                        Tg = ws.T;
                    } else if (type == BC_FLUX) {                   // imposed temperature flux, PAPER.md:435 (reading A22)
                        // reflecting velocity; the conductive flux kappa (T_ghost - T_mirror)/((2l-1) h) through
                        // the wall equals the prescribed flux F entering the domain
                        for (int e = 0; e < 3; ++e) ug[e] = (e == d) ? -ws.u[e] : ws.u[e];
                        Tg = ws.T + (2 * l - 1) * cfg.bcv[d][side] * cfg.h / cfg.kappa;
                    } else {                                        // BC_FIXED_T no-slip wall
                        for (int e = 0; e < 3; ++e) ug[e] = -ws.u[e];
                        Tg = 2.0 * cfg.bcv[d][side] - ws.T;
                    }
                    // delta = Phi_prev - Phi_ghost, Phi = -g.x (or the given potential)
                    const double delta = PhiP.empty() ? (side == 0 ? -1.0 : 1.0) * cfg.g[d] * cfg.h : PhiP[jp] - PhiP[jg];
                    // eq. (14) with p_g = rho_g T_g:  rho_g = (p_prev + 1/2 rho_prev delta)/(T_g - 1/2 delta)
                    double rg = (wp.p + 0.5 * wp.rho * delta) / (Tg - 0.5 * delta);
                    // reading A9 requires T_g > |g_d| h / 2; without it relation (14) has no positive solution and the
                    // wall closure is undefined: the ghost cell is flagged (NaN), which compute_dt reports as non-finite
                    // (only ghost cells that face interior cells: edge / corner ghosts mirror ghost cells of another
                    // wall, their doubly mirrored temperature carries no physical meaning and only their velocity is
                    // ever used, by the diagonal points of the viscous stencil)
                    bool faces_interior = true;
                    for (int e = 0; e < cfg.ndim; ++e) if (e != d && (c[e] < 0 || c[e] >= G.n[e])) faces_interior = false;
                    if (faces_interior && !(rg > 0.0)) rg = std::nan("");
                    const double pg = rg * Tg;
                    U.q[0][jg] = rg;
                    U.q[1][jg] = rg * ug[0];
                    U.q[2][jg] = rg * ug[1];
                    U.q[3][jg] = rg * ug[2];
                    U.q[4][jg] = pg / (cfg.gamma - 1.0) + 0.5 * rg * (ug[0] * ug[0] + ug[1] * ug[1] + ug[2] * ug[2]);
                }
            }
        }
    }
}

void compute_prims(const Cfg& cfg, const Grid& G, const State& U, Prim& W) {
    for (size_t j = 0; j < G.ncell; ++j) {
        const CellPrim w = cons_to_prim(cfg.gamma, U.q[0][j], U.q[1][j], U.q[2][j], U.q[3][j], U.q[4][j]);
        W.rho[j] = w.rho; W.u[0][j] = w.u[0]; W.u[1][j] = w.u[1]; W.u[2][j] = w.u[2];
        W.p[j] = w.p; W.c[j] = w.c; W.T[j] = w.T;
    }
}

// ---------------------------------------------------------------------------
// dissipative face flux (PAPER.md:44-53 tau and eta=-2/3 mu; :254-264 divergence
// form and Fourier flux; viscous stencil = reading A6).  Face normal d between
// L (index jL) and R = L + e_d.  Returns tau_{d,comp} (comp < 3) and the energy
// flux  sum_comp tau_{d,comp} * ubar_comp + kappa (T_R - T_L)/h.
// ---------------------------------------------------------------------------
void dissipative_face(const Cfg& cfg, const Grid& G, const Prim& W, int d, size_t jL,
                      double tau[3], double& fE) {
    const size_t jR = jL + G.stride(d);
    const double h = cfg.h;
    double grad[3][3];                                   // grad[e][comp] = d_e u_comp at the face
    for (int e = 0; e < 3; ++e) for (int cpn = 0; cpn < 3; ++cpn) grad[e][cpn] = 0.0;
    for (int e = 0; e < cfg.ndim; ++e) {
        const size_t se = G.stride(e);
        for (int cpn = 0; cpn < cfg.ndim; ++cpn) {
            const std::vector<double>& u = W.u[cpn];
            if (e == d) {
                grad[e][cpn] = (u[jR] - u[jL]) / h;
            } else {
                const double dL = (u[jL + se] - u[jL - se]) / (2.0 * h);
                const double dR = (u[jR + se] - u[jR - se]) / (2.0 * h);
                grad[e][cpn] = 0.5 * (dL + dR);
            }
        }
    }
    double div = 0.0;
    for (int e = 0; e < cfg.ndim; ++e) div += grad[e][e];
    fE = 0.0;
    for (int cpn = 0; cpn < 3; ++cpn) {
        tau[cpn] = 0.0;
        if (cpn >= cfg.ndim) continue;
        tau[cpn] = cfg.mu * (grad[d][cpn] + grad[cpn][d]);
        if (cpn == d) tau[cpn] += -(2.0 / 3.0) * cfg.mu * div;
        fE += tau[cpn] * (0.5 * (W.u[cpn][jL] + W.u[cpn][jR]));
    }
    fE += cfg.kappa * (W.T[jR] - W.T[jL]) / h;
}

// ---------------------------------------------------------------------------
// One full step.  form == 0: rho*E with gravity source terms (PAPER.md:194-208,
// the normative form).  form == 1: calligraphic-E form,
// eq. (11) literally with rho*calE = rho*E + rho*Phi,
// Phi = -g.x at cell centres, converted back by the relaxation Psi = Phi
// (PAPER.md:178).  The two agree to round-off (pin P4).
// form == 2: the non-conservative energy scheme of Appendix B: the same mass and momentum updates;
// the energy gets the source (dt/dx) (uS)_i, (uS)_i = 1/2 (u*_{i+1/2} S_{i+1/2} + u*_{i-1/2} S_{i-1/2}), instead of
// the mass-flux-weighted gravity work.  Reading A24: the source belongs to the acoustic sub-step (the acoustic
// energy equation of App. B carries -rho u . grad Phi), so (rho E)~ = (rho E - lam [Pi* u*] + lam (uS)_i) / L~, exactly as
// (rho u)~ carries lam S_i; summing the two sub-steps gives the update printed at PAPER.md:538.
// With cfg.phi the face potential difference is Phi_R - Phi_L of the given array instead of -g_d h.
// ---------------------------------------------------------------------------
void step(const Cfg& cfg, const Grid& G, State& U, double dt, int form) {
    const double lam = dt / cfg.h;
    const std::vector<double> PhiP = padded_potential(cfg, G);
    fill_ghosts(cfg, G, U, PhiP);

    Prim W(G.ncell);
    compute_prims(cfg, G, U, W);

    // 3. faces: arrays indexed by the L cell of each face, per axis
    std::vector<double> us[3], ps[3], Sf[3];
    for (int d = 0; d < cfg.ndim; ++d) {
        us[d].assign(G.ncell, 0.0); ps[d].assign(G.ncell, 0.0); Sf[d].assign(G.ncell, 0.0);
        const size_t sd = G.stride(d);
        const double gh = cfg.g[d] * cfg.h;
        int c[3];
        for (c[2] = -G.off[2]; c[2] < G.n[2] + G.off[2]; ++c[2])
        for (c[1] = -G.off[1]; c[1] < G.n[1] + G.off[1]; ++c[1])
        for (c[0] = -G.off[0]; c[0] < G.n[0] + G.off[0]; ++c[0]) {
            if (c[d] + 1 >= G.n[d] + G.off[d]) continue;       // no R cell
            const size_t jL = G.at(c), jR = jL + sd;
            // S_{i+1/2} = -1/2 (rho_i + rho_{i+1}) (Phi_{i+1} - Phi_i): "gh" = -(Phi_R - Phi_L)
            const double ghf = PhiP.empty() ? gh : -(PhiP[jR] - PhiP[jL]);
            const Face f = acoustic_face(W.rho[jL], W.u[d][jL], W.p[jL], W.c[jL],
                                         W.rho[jR], W.u[d][jR], W.p[jR], W.c[jR], ghf, cfg.theta);
            us[d][jL] = f.ustar; ps[d][jL] = f.pistar; Sf[d][jL] = f.S;
        }
    }

    // potential at cell centres (only used by form 1)
    auto Phi = [&](int i, int j, int k) {
        if (!PhiP.empty()) return PhiP[G.at(i, j, k)];
        return -(cfg.g[0] * (i + 0.5) * cfg.h + cfg.g[1] * (j + 0.5) * cfg.h + cfg.g[2] * (k + 0.5) * cfg.h);
    };

    // 4. acoustic update on interior + 1 ring (multi-D unsplit, reading A1)
    State Ut(G.ncell);
    {
        int c[3], lo[3], hi[3];
        for (int e = 0; e < 3; ++e) { lo[e] = e < cfg.ndim ? -1 : 0; hi[e] = e < cfg.ndim ? G.n[e] + 1 : G.n[e]; }
        for (c[2] = lo[2]; c[2] < hi[2]; ++c[2])
        for (c[1] = lo[1]; c[1] < hi[1]; ++c[1])
        for (c[0] = lo[0]; c[0] < hi[0]; ++c[0]) {
            const size_t j = G.at(c);
            double sum_du = 0.0, sum_dpu = 0.0, sum_uS = 0.0;
            double mom[3] = {U.q[1][j], U.q[2][j], U.q[3][j]};
            for (int d = 0; d < cfg.ndim; ++d) {
                const size_t jm = j - G.stride(d);               // face d- is indexed by its L cell
                sum_du  += us[d][j] - us[d][jm];                                  // [u*]
                sum_dpu += ps[d][j] * us[d][j] - ps[d][jm] * us[d][jm];           // [Pi* u*]
                const double Si = 0.5 * (Sf[d][j] + Sf[d][jm]);                   // S_i
                mom[d] = mom[d] - lam * (ps[d][j] - ps[d][jm]) + lam * Si;
                sum_uS += 0.5 * (us[d][j] * Sf[d][j] + us[d][jm] * Sf[d][jm]);    // (uS)_i, PAPER.md:544 (App. B)
            }
            const double Lt = 1.0 + lam * sum_du;                                 // L~
            double En = U.q[4][j];
            if (form == 1) En += U.q[0][j] * Phi(c[0], c[1], c[2]);               // rho*calE
            Ut.q[0][j] = U.q[0][j] / Lt;
            Ut.q[1][j] = mom[0] / Lt;
            Ut.q[2][j] = mom[1] / Lt;
            Ut.q[3][j] = mom[2] / Lt;
            if (form == 2) En += lam * sum_uS;                                    // App. B, reading A24
            Ut.q[4][j] = (En - lam * sum_dpu) / Lt;                               // reading A3: divided by L~
        }
    }

    // 5. transport + dissipative fluxes + conservative update on the interior
    State Un(G.ncell);
    const bool dissip = (cfg.mu > 0.0) || (cfg.kappa > 0.0);
    {
        int c[3];
        for (c[2] = 0; c[2] < G.n[2]; ++c[2])
        for (c[1] = 0; c[1] < G.n[1]; ++c[1])
        for (c[0] = 0; c[0] < G.n[0]; ++c[0]) {
            const size_t j = G.at(c);
            double dF[5] = {0, 0, 0, 0, 0};      // sum_d (flux_{d+} - flux_{d-})
            double src[5] = {0, 0, 0, 0, 0};
            for (int d = 0; d < cfg.ndim; ++d) {
                const size_t sd = G.stride(d);
                double Fs[2][5];                 // [0]: face d- ; [1]: face d+
                for (int side = 0; side < 2; ++side) {
                    const size_t jL = side == 0 ? j - sd : j;
                    const size_t jR = jL + sd;
                    const double ustar = us[d][jL], pistar = ps[d][jL];
                    const size_t jup = (ustar >= 0.0) ? jL : jR;      // PAPER.md:174, reading A10
                    double F[5];
                    for (int f = 0; f < 5; ++f) F[f] = Ut.q[f][jup] * ustar;      // [b~ u*]
                    F[1 + d] += pistar;                                           // + Pi* on the normal momentum
                    F[4] += pistar * ustar;                                       // (E~ + Pi*) u*
                    if (form == 1) {
                        // eq. (11) is used as printed: nothing else to add
                    } else if (form == 2) {
                        // App. B: the energy source is lam (uS)_i, added once per axis below
                    } else if (!PhiP.empty()) {
                        // the same gravity work with a general potential: -lam ( m_+ (Phi_up+ - Phi_i) - m_- (Phi_up- - Phi_i) ),
                        // Phi_up = Phi of the upwind cell: only inflow faces contribute, with -(Phi_R - Phi_L) of that face
                        const double m = Ut.q[0][jup] * ustar;
                        const double ghf = -(PhiP[jR] - PhiP[jL]);
                        if (side == 1) src[4] += lam * ghf * std::min(m, 0.0);
                        else           src[4] += lam * ghf * std::max(m, 0.0);
                    } else {
                        // gravity work  -dt {rho u d_x Phi}_i = -lam( [rho~ u* Phi] - [rho~ u*] Phi_i )
                        // with Phi_face = Phi_upwind (reading A13):
                        //   face d+ contributes dt*g_d*min(m,0), face d- contributes dt*g_d*max(m,0)
                        const double m = Ut.q[0][jup] * ustar;
                        if (side == 1) src[4] += dt * cfg.g[d] * std::min(m, 0.0);
                        else           src[4] += dt * cfg.g[d] * std::max(m, 0.0);
                    }
                    if (dissip) {
                        double tau[3], fE;
                        dissipative_face(cfg, G, W, d, jL, tau, fE);
                        for (int e = 0; e < 3; ++e) F[1 + e] -= tau[e];
                        F[4] -= fE;
                    }
                    for (int f = 0; f < 5; ++f) Fs[side][f] = F[f];
                }
                for (int f = 0; f < 5; ++f) dF[f] += Fs[1][f] - Fs[0][f];
                src[1 + d] += lam * (0.5 * (Sf[d][j] + Sf[d][j - sd]));           // + lam * S_i
                if (form == 2) src[4] += lam * (0.5 * (us[d][j] * Sf[d][j] + us[d][j - sd] * Sf[d][j - sd]));   // + lam (uS)_i
            }
            double old[5];
            for (int f = 0; f < 5; ++f) old[f] = U.q[f][j];
            if (form == 1) old[4] += U.q[0][j] * Phi(c[0], c[1], c[2]);
            double nw[5];
            for (int f = 0; f < 5; ++f) nw[f] = old[f] - lam * dF[f] + src[f];
            if (form == 1) nw[4] -= nw[0] * Phi(c[0], c[1], c[2]);                // relaxation Psi = Phi
            for (int f = 0; f < 5; ++f) Un.q[f][j] = nw[f];
        }
    }
    for (int f = 0; f < 5; ++f) U.q[f].swap(Un.q[f]);
    // (ghosts of the new state are stale; they are refilled at the start of the next step)
}

// 6. CFL (reading A4): dt = cfl / max_c [ sum_d (|u_d| + c)/h + 2 ndim max(4mu/3,(gamma-1)kappa)/(rho h^2) ]
double max_rate(const Cfg& cfg, const Grid& G, const State& U) {
    double mx = 0.0;
    bool bad = false;
    int c[3];
    for (c[2] = 0; c[2] < G.n[2]; ++c[2])
    for (c[1] = 0; c[1] < G.n[1]; ++c[1])
    for (c[0] = 0; c[0] < G.n[0]; ++c[0]) {
        const size_t j = G.at(c);
        const CellPrim w = cons_to_prim(cfg.gamma, U.q[0][j], U.q[1][j], U.q[2][j], U.q[3][j], U.q[4][j]);
        double r = 0.0;
        for (int d = 0; d < cfg.ndim; ++d) r += (std::fabs(w.u[d]) + w.c) / cfg.h;
        const double D = std::max(4.0 * cfg.mu / 3.0, (cfg.gamma - 1.0) * cfg.kappa);
        r += 2.0 * cfg.ndim * D / (w.rho * cfg.h * cfg.h);
        if (!(r == r) || std::isinf(r)) bad = true;
        if (r > mx) mx = r;
    }
    return bad ? std::nan("") : mx;
}

// dense interior-only arrays (x fastest) <-> padded state
void load_dense(const Grid& G, State& U, const double* const in[5]) {
    for (int f = 0; f < 5; ++f) {
        if (!in[f]) continue;
        size_t s = 0;
        for (int k = 0; k < G.n[2]; ++k) for (int j = 0; j < G.n[1]; ++j) for (int i = 0; i < G.n[0]; ++i)
            U.q[f][G.at(i, j, k)] = in[f][s++];
    }
}
void store_dense(const Grid& G, const State& U, double* const out[5]) {
    for (int f = 0; f < 5; ++f) {
        if (!out[f]) continue;
        size_t s = 0;
        for (int k = 0; k < G.n[2]; ++k) for (int j = 0; j < G.n[1]; ++j) for (int i = 0; i < G.n[0]; ++i)
            out[f][s++] = U.q[f][G.at(i, j, k)];
    }
}

Cfg make_cfg(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
             int theta, const int* bc_type, const double* bc_val, const double* phi = nullptr) {
    Cfg c;
    c.phi = phi;
    c.n[0] = nx; c.n[1] = ny; c.n[2] = nz;
    c.ndim = nz == 1 ? 2 : 3;
    c.h = h; c.gamma = gamma; c.mu = mu; c.kappa = kappa; c.theta = theta;
    for (int d = 0; d < 3; ++d) {
        c.g[d] = g[d];
        for (int s = 0; s < 2; ++s) { c.bc[d][s] = bc_type[2 * d + s]; c.bcv[d][s] = bc_val[2 * d + s]; }
    }
    return c;
}

}  // namespace

// ---------------------------------------------------------------------------
// C entry points for ctypes (oracle/ark_oracle.py).  All pointers are HOST.
// State arrays are dense interior-only nx*ny*nz, x fastest; rhow may be NULL
// when nz == 1.  bc_type / bc_val are [x_lo, x_hi, y_lo, y_hi, z_lo, z_hi].
// ---------------------------------------------------------------------------
extern "C" {

double oracle_K(void) { return K_IMP; }

// Advance nsteps.  If dts != NULL it holds nsteps prescribed time steps; otherwise each
// dt = cfl / max_rate (and, if dts_out != NULL, is recorded there).  form: 0 = E + source
// (normative), 1 = eq. (11).  Returns 0, or -4 if a non-finite rate was met.
// (2 = Appendix B).  phi: optional dense potential at the cell centres (NULL: constant g).
int oracle_run_phi(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
                   int theta, const int* bc_type, const double* bc_val,
                   double* rho, double* rhou, double* rhov, double* rhow, double* E,
                   int nsteps, double cfl, const double* dts, double* dts_out, int form, const double* phi);

int oracle_run(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
               int theta, const int* bc_type, const double* bc_val,
               double* rho, double* rhou, double* rhov, double* rhow, double* E,
               int nsteps, double cfl, const double* dts, double* dts_out, int form) {
    return oracle_run_phi(nx, ny, nz, h, gamma, g, mu, kappa, theta, bc_type, bc_val, rho, rhou, rhov, rhow, E, nsteps, cfl, dts,
                          dts_out, form, nullptr);
}

int oracle_run_phi(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
                   int theta, const int* bc_type, const double* bc_val,
                   double* rho, double* rhou, double* rhov, double* rhow, double* E,
                   int nsteps, double cfl, const double* dts, double* dts_out, int form, const double* phi) {
    const Cfg cfg = make_cfg(nx, ny, nz, h, gamma, g, mu, kappa, theta, bc_type, bc_val, phi);
    const Grid G(cfg);
    State U(G.ncell);
    const double* in[5] = {rho, rhou, rhov, rhow, E};
    load_dense(G, U, in);
    for (int s = 0; s < nsteps; ++s) {
        double dt;
        if (dts) dt = dts[s];
        else {
            const double r = max_rate(cfg, G, U);
            if (!(r > 0.0) || std::isinf(r)) return -4;
            dt = cfl / r;
        }
        if (dts_out) dts_out[s] = dt;
        step(cfg, G, U, dt, form);
    }
    double* out[5] = {rho, rhou, rhov, rhow, E};
    store_dense(G, U, out);
    return 0;
}

// max_c rate_c of reading A4 (NaN if any cell's rate is non-finite).
double oracle_max_rate(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
                       int theta, const int* bc_type, const double* bc_val,
                       const double* rho, const double* rhou, const double* rhov, const double* rhow, const double* E) {
    const Cfg cfg = make_cfg(nx, ny, nz, h, gamma, g, mu, kappa, theta, bc_type, bc_val);
    const Grid G(cfg);
    State U(G.ncell);
    const double* in[5] = {rho, rhou, rhov, rhow, E};
    load_dense(G, U, in);
    return max_rate(cfg, G, U);
}

// Ghost fill only: returns the PADDED arrays ((nx+4)*(ny+4)*(nz+4 or 1), x fastest) for BC tests.
int oracle_fill_ghosts(int nx, int ny, int nz, double h, double gamma, const double* g, double mu, double kappa,
                       int theta, const int* bc_type, const double* bc_val,
                       const double* rho, const double* rhou, const double* rhov, const double* rhow, const double* E,
                       double* prho, double* prhou, double* prhov, double* prhow, double* pE) {
    const Cfg cfg = make_cfg(nx, ny, nz, h, gamma, g, mu, kappa, theta, bc_type, bc_val);
    const Grid G(cfg);
    State U(G.ncell);
    const double* in[5] = {rho, rhou, rhov, rhow, E};
    load_dense(G, U, in);
    fill_ghosts(cfg, G, U, padded_potential(cfg, G));
    double* out[5] = {prho, prhou, prhov, prhow, pE};
    for (int f = 0; f < 5; ++f) if (out[f]) std::memcpy(out[f], U.q[f].data(), G.ncell * sizeof(double));
    return 0;
}

// Diagnostics the paper reports (PAPER.md:398-407 maximum velocity, :435 mean absolute velocity, :14 mass and total
// energy).  out = { max |u|, mean |u|, sum 1/2 rho |u|^2 dV, max |u|/c, sum rho dV, sum (E + rho Phi) dV },
// Phi = -g.x at the cell centres, dV = h^ndim.  Plain loops, long double accumulators.
void oracle_diagnostics(int nx, int ny, int nz, double h, double gamma, const double* g,
                        const double* rho, const double* rhou, const double* rhov, const double* rhow, const double* E,
                        double* out) {
    const int ndim = nz == 1 ? 2 : 3;
    long double s_speed = 0, s_ke = 0, s_m = 0, s_e = 0;
    double max_speed = 0.0, max_mach = 0.0;
    size_t j = 0;
    for (int k = 0; k < nz; ++k) for (int jy = 0; jy < ny; ++jy) for (int i = 0; i < nx; ++i, ++j) {
        const double mz = (ndim == 3 && rhow) ? rhow[j] : 0.0;
        const CellPrim w = cons_to_prim(gamma, rho[j], rhou[j], rhov[j], mz, E[j]);
        const double speed = std::sqrt(w.u[0] * w.u[0] + w.u[1] * w.u[1] + w.u[2] * w.u[2]);
        const double phi = -(g[0] * (i + 0.5) * h + g[1] * (jy + 0.5) * h + (ndim == 3 ? g[2] * (k + 0.5) * h : 0.0));
        max_speed = std::max(max_speed, speed);
        max_mach = std::max(max_mach, speed / w.c);
        s_speed += speed;
        s_ke += 0.5 * w.rho * speed * speed;
        s_m += w.rho;
        s_e += E[j] + w.rho * phi;
    }
    const double vol = ndim == 3 ? h * h * h : h * h;
    out[0] = max_speed;
    out[1] = (double)(s_speed / (long double)((size_t)nx * ny * nz));
    out[2] = (double)(s_ke * vol);
    out[3] = max_mach;
    out[4] = (double)(s_m * vol);
    out[5] = (double)(s_e * vol);
}

// One acoustic face from primitive L/R data (pin P8).  out = {cL, cR, a, S, u*, theta, Pi*}.
void oracle_face(double gamma, double rhoL, double unL, double pL, double rhoR, double unR, double pR,
                 double gh, int theta_flag, double* out) {
    const double cL = std::sqrt(gamma * pL / rhoL), cR = std::sqrt(gamma * pR / rhoR);
    const Face f = acoustic_face(rhoL, unL, pL, cL, rhoR, unR, pR, cR, gh, theta_flag);
    out[0] = cL; out[1] = cR; out[2] = f.a; out[3] = f.S; out[4] = f.ustar; out[5] = f.theta; out[6] = f.pistar;
}

}  // extern "C"
