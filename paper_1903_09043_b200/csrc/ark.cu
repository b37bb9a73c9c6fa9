// ark.cu -- C-ABI implementation (include/ark.h) on top of the sm_100a kernels in ark_device.cuh / ark_step.cuh.
// No torch types, no CPU fallback: every step of the hot path runs in the kernels of this library.
#include "../../include/ark.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <vector>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ark_step3d.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, const char* a = "", long long b = 0) {
    snprintf(g_err, sizeof g_err, fmt, a, b);
    return code;
}
#define ARK_CUDA(call)                                                             \
    do {                                                                           \
        cudaError_t e_ = (call);                                                   \
        if (e_ != cudaSuccess) return fail(ARK_ECUDA, "CUDA error: %s (%lld)", cudaGetErrorString(e_), (long long)__LINE__); \
    } while (0)

// tile of the fused step kernel
constexpr int TX3 = ARK_TX3, NW3 = ARK_NW3;   // 3D: outputs per row, row pairs per block
constexpr int TY3 = 2 * NW3 - 4;
constexpr int TX2 = ARK_TX2, TY2 = ARK_TY2;   // 2D

#define ARK_KERNEL_REV "r2.6"
constexpr int CFL_BLOCK = 256;
#define ARK_MAX_TIMED 4096
constexpr int MAX_SCRATCH = 1 << 16;          // per-block rate slots
constexpr int DIAG_BLOCKS = 1184;             // ark_diagnostics: partials live in the last DIAG_BLOCKS * 6 rate slots

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
    int px, py, pz, offz, nf;
    long long fstride;       // doubles
    size_t state_bytes;      // one padded state (nf fields)
    size_t scratch_off, result_off, dtlog_off, stage_off, total;
};

bool valid_sizes(int nx, int ny, int nz) {
    return nx >= 4 && ny >= 4 && (nz == 1 || nz >= 4) && nx <= (1 << 14) && ny <= (1 << 14) && nz <= (1 << 14);
}

constexpr int DTLOG_MAX = 1 << 16;

Layout make_layout(int nx, int ny, int nz) {
    Layout L;
    const bool d3 = nz > 1;
    L.nf = d3 ? 5 : 4;
    L.offz = d3 ? ARK_NG : 0;
    L.px = (int)round_up((size_t)nx + ARK_XOFF + ARK_NG, 16);
    L.py = ny + 2 * ARK_NG;
    L.pz = d3 ? nz + 2 * ARK_NG : 1;
    L.fstride = (long long)round_up((size_t)L.px * L.py * L.pz, 32);
    L.state_bytes = (size_t)L.nf * L.fstride * sizeof(double);
    size_t off = 2 * L.state_bytes;
    L.scratch_off = off; off += round_up((size_t)MAX_SCRATCH * sizeof(double), 256);
    L.result_off = off;  off += 256;
    L.dtlog_off = off;   off += round_up((size_t)DTLOG_MAX * sizeof(double), 256);
    L.stage_off = off;   off += round_up((size_t)nx * ny * nz * sizeof(double), 256);   // one dense field (host copies)
    L.total = off;
    return L;
}

}  // namespace

struct ark_solver {
    ArkParams P;
    Layout L;
    char* ws;
    double* U[2];           // padded states; U[cur] holds the current one
    int cur;
    double* scratch;        // per-block rates
    double* result;         // [0] max rate, [1] dt
    double* dtlog;
    double* stage;
    cudaStream_t stream;
    int rate_slots;         // >0: scratch[0..rate_slots) holds the per-block rates of the CURRENT state
    bool xghost_valid;      // periodic x: the step kernel already wrote the x ghost columns of the current state
    bool xyghost_valid;     // the x and y ghost sweeps already ran on the current state (ark_get_halo)
    bool yghost_valid;      // 2D, periodic x and y: the step kernel already wrote the y ghost rows (and corners) as well
    dim3 step_grid;
    int zchunk;
    long long launches;
    CUtensorMap tmap[2];    // 3D: tensor maps of the two padded states (TMA tile loads of the step kernel)
    // ark_run: two consecutive steps (A->B, B->A) captured once as a CUDA graph and replayed (the small 2D configs are
    // launch-latency-bound: 5 launches per step).  Capture needs a non-legacy stream of the library's own.
    cudaStream_t gstream;
    cudaEvent_t gev_in, gev_out;
    cudaGraphExec_t gexec;
    int g_cur, g_log;       // state the cached graph was captured for: buffer parity, with / without dt log
    double g_cfl;
    long long g_launches;   // kernel launches inside one replay
    double* h_pinned;       // 2 doubles, pinned, for the 16-byte D2H of compute_dt
    int device;             // the CUDA device the handle was created on (entry points check it is current)
    // optional event bracketing of the step kernel (measurement hook): allocated on first use, outside the handle
    bool timing;
    int n_timed;
    struct ArkTimer* timer;
};

struct ArkTimer { cudaEvent_t ev0[ARK_MAX_TIMED], ev1[ARK_MAX_TIMED]; };

namespace {

// Tensor map of one padded 3D state for the step kernel's TMA loads: 4-D tensor (x, y, z, field) of fp64, box =
// (RX columns, RY rows, 1 plane, 5 fields), no swizzle, zero fill outside the array (ragged tiles).  The encoder is a
// driver entry point fetched through the runtime, so the library does not link libcuda.
int make_tensor_map(CUtensorMap* out, const Layout& L, double* base, int rx, int ry) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        ARK_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) return fail(ARK_ECUDA, "cuTensorMapEncodeTiled is not available%s");
        encode = (encode_fn)fn;
    }
    const cuuint64_t dims[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)L.pz, (cuuint64_t)L.nf};
    const cuuint64_t strides[3] = {(cuuint64_t)L.px * 8, (cuuint64_t)L.px * L.py * 8, (cuuint64_t)L.fstride * 8};
    const cuuint32_t box[4] = {(cuuint32_t)rx, (cuuint32_t)ry, 1, (cuuint32_t)L.nf};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ARK_ECUDA, "cuTensorMapEncodeTiled failed (%s%lld)", "", (long long)r);
    return ARK_OK;
}

// every entry point runs on the device the handle was created on
int check_device(const ark_solver* s) {
    int dev = -1;
    ARK_CUDA(cudaGetDevice(&dev));
    if (dev != s->device) return fail(ARK_EINVAL, "the solver was created on CUDA device %s%lld, which is not the current device", "", (long long)s->device);
    return ARK_OK;
}
#define ARK_ON_DEVICE(s) do { const int rc_ = check_device(s); if (rc_ != ARK_OK) return rc_; } while (0)

int grid_for(long long n, int block, int cap = 148 * 8) {
    long long b = (n + block - 1) / block;
    if (b < 1) b = 1;
    return (int)(b < cap ? b : cap);
}

template <bool VISC, bool GEN>
int launch_step2(ark_solver* s, double dt, const double* dt_dev) {
    using C = ArkStepCfg<2, VISC, TX2, TY2>;
    auto kern = ark_k_step<2, VISC, GEN, TX2, TY2>;
    const bool timed = s->timing && s->n_timed < ARK_MAX_TIMED;
    if (timed) ARK_CUDA(cudaEventRecord(s->timer->ev0[s->n_timed], s->stream));
    kern<<<s->step_grid, C::NT, C::SMEM_BYTES, s->stream>>>(s->P, s->U[s->cur], s->U[1 - s->cur], dt, dt_dev, s->scratch);
    if (timed) { ARK_CUDA(cudaEventRecord(s->timer->ev1[s->n_timed], s->stream)); s->n_timed++; }
    ARK_CUDA(cudaGetLastError());
    s->launches++;
    return ARK_OK;
}

// x and y sweeps of the ghost fill (interior z range); the z sweep covers the extended x, y range afterwards
int launch_bc_xy(ark_solver* s, double* U) {
    const ArkParams& P = s->P;
    if (s->xyghost_valid) return ARK_OK;
    if (P.bc[0][0] == ARK_BCK_PERIODIC) {
        // (the fused step kernels write the periodic x ghost columns of the state they produce; the sweep is only
        // needed for a state that came from outside)
        if (!s->xghost_valid) {
            const long long n = 2LL * P.ny * P.nz * P.nf;
            ark_k_bc_x_periodic<<<grid_for(n, 256, 148 * 16), 256, 0, s->stream>>>(P, U);
            s->launches++;
        }
    } else {
        const long long n = 2LL * P.ny * P.nz;
        ark_k_bc<0><<<grid_for(n, 128), 128, 0, s->stream>>>(P, U);
        s->launches++;
    }
    if (!s->yghost_valid) {
        const long long n = 2LL * (P.nx + 2 * ARK_NG) * P.nz;
        ark_k_bc<1><<<grid_for(n, 128), 128, 0, s->stream>>>(P, U);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

int launch_bc(ark_solver* s, double* U) {
    const ArkParams& P = s->P;
    const int rc = launch_bc_xy(s, U);
    if (rc != ARK_OK) return rc;
    if (P.ndim == 3 && !(P.bc[2][0] == ARK_BCK_EXTERNAL && P.bc[2][1] == ARK_BCK_EXTERNAL)) {
        const long long n = 2LL * (P.nx + 2 * ARK_NG) * (P.ny + 2 * ARK_NG);
        ark_k_bc<2><<<grid_for(n, 128), 128, 0, s->stream>>>(P, U);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

template <bool VISC, bool GXY, bool GEN>
int launch_step3(ark_solver* s, double dt, const double* dt_dev) {
    using C = ArkCfg3<VISC, TX3, NW3>;
    auto kern = ark_k_step3<VISC, GXY, GEN, TX3, NW3>;
    const bool timed = s->timing && s->n_timed < ARK_MAX_TIMED;
    if (timed) ARK_CUDA(cudaEventRecord(s->timer->ev0[s->n_timed], s->stream));
    kern<<<s->step_grid, C::NT, C::SMEM_BYTES, s->stream>>>(s->P, s->U[s->cur], s->U[1 - s->cur], dt, dt_dev,
                                                            s->scratch, s->zchunk, s->tmap[s->cur]);
    if (timed) { ARK_CUDA(cudaEventRecord(s->timer->ev1[s->n_timed], s->stream)); s->n_timed++; }
    ARK_CUDA(cudaGetLastError());
    s->launches++;
    return ARK_OK;
}

// opt-in to the large dynamic shared memory of the step kernels on the CURRENT device (the attribute is per device)
template <typename K>
int set_smem(K kern, size_t bytes) {
    ARK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return ARK_OK;
}
int set_step_attributes(int ndim) {
    int rc = ARK_OK;
    if (ndim == 3) {
        const size_t bv = ArkCfg3<true, TX3, NW3>::SMEM_BYTES, bi = ArkCfg3<false, TX3, NW3>::SMEM_BYTES;
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<true, true, false, TX3, NW3>, bv);
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<true, false, false, TX3, NW3>, bv);
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<true, true, true, TX3, NW3>, bv);
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<false, true, false, TX3, NW3>, bi);
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<false, false, false, TX3, NW3>, bi);
        if (rc == ARK_OK) rc = set_smem(ark_k_step3<false, true, true, TX3, NW3>, bi);
    } else {
        const size_t bv = ArkStepCfg<2, true, TX2, TY2>::SMEM_BYTES, bi = ArkStepCfg<2, false, TX2, TY2>::SMEM_BYTES;
        if (rc == ARK_OK) rc = set_smem(ark_k_step<2, true, false, TX2, TY2>, bv);
        if (rc == ARK_OK) rc = set_smem(ark_k_step<2, true, true, TX2, TY2>, bv);
        if (rc == ARK_OK) rc = set_smem(ark_k_step<2, false, false, TX2, TY2>, bi);
        if (rc == ARK_OK) rc = set_smem(ark_k_step<2, false, true, TX2, TY2>, bi);
    }
    return rc;
}

int do_step(ark_solver* s, double dt, const double* dt_dev) {
    int rc = launch_bc(s, s->U[s->cur]);
    if (rc != ARK_OK) return rc;
    const bool visc = s->P.mu > 0.0 || s->P.kappa > 0.0;
    const bool gen = s->P.phi != nullptr || s->P.eform != 0;    // general path: array-valued potential and / or Appendix B
    if (s->P.ndim == 3) {
        const bool gxy = s->P.D.g_on[0] || s->P.D.g_on[1];
        if (gen)       rc = visc ? launch_step3<true, true, true>(s, dt, dt_dev) : launch_step3<false, true, true>(s, dt, dt_dev);
        else if (visc) rc = gxy ? launch_step3<true, true, false>(s, dt, dt_dev) : launch_step3<true, false, false>(s, dt, dt_dev);
        else           rc = gxy ? launch_step3<false, true, false>(s, dt, dt_dev) : launch_step3<false, false, false>(s, dt, dt_dev);
    } else {
        if (gen) rc = visc ? launch_step2<true, true>(s, dt, dt_dev) : launch_step2<false, true>(s, dt, dt_dev);
        else     rc = visc ? launch_step2<true, false>(s, dt, dt_dev) : launch_step2<false, false>(s, dt, dt_dev);
    }
    if (rc != ARK_OK) return rc;
    s->cur = 1 - s->cur;
    s->xghost_valid = s->P.bc[0][0] == ARK_BCK_PERIODIC;
    s->yghost_valid = s->P.ndim == 2 && s->xghost_valid && s->P.bc[1][0] == ARK_BCK_PERIODIC;
    s->xyghost_valid = false;
    s->rate_slots = (int)(s->step_grid.x * s->step_grid.y * s->step_grid.z);   // fused CFL epilogue filled them
    return ARK_OK;
}

// max rate of the current state -> result[0], dt -> result[1] (device).  Uses the step kernel's epilogue
// values when they describe the current state, otherwise runs the standalone pass 1.
int reduce_rate(ark_solver* s, double cfl, double* dt_log) {
    int nvals = s->rate_slots;
    if (nvals <= 0) {
        const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
        nvals = grid_for(n, CFL_BLOCK, 148 * 8);
        ark_k_cfl_pass1<<<nvals, CFL_BLOCK, 0, s->stream>>>(s->P, s->U[s->cur], s->scratch);
        s->launches++;
        s->rate_slots = nvals;
    }
    ark_k_cfl_pass2<<<1, 1024, 0, s->stream>>>(s->scratch, nvals, cfl, s->result, dt_log, (int*)(s->result + 4));
    s->launches++;
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

}  // namespace

extern "C" {

const char* ark_last_error(void) { return g_err; }

const char* ark_version_string(void) {
    static char buf[256];
    // ARK_KERNEL_REV names the revision of the 3D step kernel (ark_k_step3) the committed ncu counters (profiles/) belong
    // to: bump it with every change to THAT kernel's arithmetic or memory traffic (the 2D kernel has no committed counters;
    // its changes are recorded in DESIGN.md 5.3 only)
    snprintf(buf, sizeof buf, "ark-b200 0.2 (sm_100a; K=%.2f; ng=%d; tile3d=%dx%d (%d row pairs) tile2d=%dx%d; kernels %s)", ARK_K_IMPEDANCE, ARK_NG,
             TX3, TY3, NW3, TX2, TY2, ARK_KERNEL_REV);
    return buf;
}

}  // extern "C"

namespace {

// Time (in plane iterations) the grid of the 3D step kernel takes when its blocks are handed out in blockIdx order (x, y,
// then z chunk) to nsm SMs, one block per SM, each block costing its planes + ~2.5 planes of prologue.
constexpr double g_chunk_ovh = 2.5;                           // prologue of a chunk in plane iterations (fitted, profiles/r02_step_kernel.md)
double chunk_makespan(long long ncol, const int* chunk, int nchunk, int nsm) {
    std::vector<double> heap((size_t)nsm, 0.0);               // min-heap of the SMs' finish times
    auto cmp = [](double a, double b) { return a > b; };
    for (int c = 0; c < nchunk; ++c)
        for (long long b = 0; b < ncol; ++b) {
            std::pop_heap(heap.begin(), heap.end(), cmp);
            heap.back() += chunk[c] + g_chunk_ovh;
            std::push_heap(heap.begin(), heap.end(), cmp);
        }
    return *std::max_element(heap.begin(), heap.end());
}

// z chunks of the 3D step kernel.  They exist only to create blocks; every chunk costs a 2-plane prologue, and the last
// wave of blocks leaves SMs idle.  Chunk sizes that DECREASE geometrically (large chunks first, small ones to fill the
// tail) beat uniform ones (simulated: 256^3 310 -> 295 plane iterations per SM, 512^3 2195 -> 2154): candidates =
// nchunk 1..16 x ratio 1 .. 0.4, scored by the scheduling simulation above.  zb[0..nchunk] = chunk boundaries.
int choose_zchunks(int nx, int ny, int nz, int nsm, int* zb) {
    const long long ncol = (long long)((nx + TX3 - 1) / TX3) * ((ny + TY3 - 1) / TY3);
    const double ratios[7] = {1.0, 0.9, 0.8, 0.7, 0.6, 0.5, 0.4};
    int best[ARK_MAX_ZCHUNKS] = {nz}, nbest = 1;
    double best_t = 1e300;
    const bool big = ncol * ARK_MAX_ZCHUNKS > 50000;            // huge grids: many waves anyway, skip the simulation
    for (int n = 1; n <= ARK_MAX_ZCHUNKS && n * 4 <= nz; ++n) {
        if (n > 1 && ncol * n > MAX_SCRATCH - DIAG_BLOCKS * ARK_NDIAG) break;       // one CFL rate slot per block
        for (int ir = 0; ir < 7; ++ir) {
            int ch[ARK_MAX_ZCHUNKS];
            double w = 1.0, sum = 0.0;
            for (int i = 0; i < n; ++i) { sum += w; w *= ratios[ir]; }
            w = 1.0;
            int tot = 0;
            for (int i = 0; i < n; ++i) { ch[i] = (int)std::floor(nz * w / sum + 0.5); if (ch[i] < 4) ch[i] = 4; tot += ch[i]; w *= ratios[ir]; }
            ch[0] += nz - tot;
            if (ch[0] < 4 || (n > 1 && ch[0] < ch[1])) continue;
            const double t = big ? (double)((ncol * n + nsm - 1) / nsm) * (nz / (double)n + g_chunk_ovh) : chunk_makespan(ncol, ch, n, nsm);
            if (t < best_t) { best_t = t; nbest = n; for (int i = 0; i < n; ++i) best[i] = ch[i]; }
            if (n == 1 || big) break;
        }
    }
    // hill climb from the best geometric candidate: move a few planes from one chunk to another while the simulated
    // makespan drops
    if (!big && nbest > 1) {
        bool improved = true;
        for (int round = 0; improved && round < 40; ++round) {
            improved = false;
            for (int i = 0; i < nbest; ++i)
                for (int j = 0; j < nbest; ++j) {
                    if (i == j) continue;
                    for (int d = 8; d >= 1; d >>= 1) {
                        if (best[i] - d < 4) continue;
                        best[i] -= d; best[j] += d;
                        const double t = chunk_makespan(ncol, best, nbest, nsm);
                        if (t < best_t - 1e-9) { best_t = t; improved = true; }
                        else { best[i] += d; best[j] -= d; }
                    }
                }
        }
    }
    zb[0] = 0;
    for (int i = 0; i < nbest; ++i) zb[i + 1] = zb[i] + best[i];
    return nbest;
}

// number of blocks of the fused step kernel (= per-block CFL rate slots it fills)
long long step_blocks(int nx, int ny, int nz, dim3* grid, int* zb, int nsm = 148) {
    if (nz > 1) {
        const int gx = (nx + TX3 - 1) / TX3, gy = (ny + TY3 - 1) / TY3;
        int tmp[ARK_MAX_ZCHUNKS + 1];
        const int nchunk = choose_zchunks(nx, ny, nz, nsm, zb ? zb : tmp);
        if (grid) *grid = dim3(gx, gy, nchunk);
        return (long long)gx * gy * nchunk;
    }
    const int gx = (nx + TX2 - 1) / TX2, gy = (ny + TY2 - 1) / TY2;
    if (grid) *grid = dim3(gx, gy, 1);
    return (long long)gx * gy;
}

// Cheap (the size queries ark_workspace_bytes / ark_potential_bytes / ark_halo_bytes go through it; the scheduling
// simulation of choose_zchunks costs milliseconds and runs in ark_create only): choose_zchunks never takes more chunks
// than the rate scratch has slots for and a single chunk is always allowed, so the grid fits exactly when its columns do.
bool supported_grid(int nx, int ny, int nz) {
    if (!valid_sizes(nx, ny, nz)) return false;
    const long long ncol = nz > 1 ? (long long)((nx + TX3 - 1) / TX3) * ((ny + TY3 - 1) / TY3)
                                  : (long long)((nx + TX2 - 1) / TX2) * ((ny + TY2 - 1) / TY2);
    return ncol <= MAX_SCRATCH - DIAG_BLOCKS * ARK_NDIAG;
}

}  // namespace

extern "C" {

size_t ark_workspace_bytes(int nx, int ny, int nz) {
    if (!supported_grid(nx, ny, nz)) return 0;
    return make_layout(nx, ny, nz).total;
}

int ark_create(ark_solver** out, int nx, int ny, int nz, double dx, double gamma, const double g[3], double mu,
               double kappa, int low_mach_theta, const ark_bc* bc, void* d_workspace, size_t workspace_bytes,
               void* cuda_stream) {
    if (!out) return fail(ARK_EINVAL, "ark_create: out is NULL%s");
    *out = nullptr;
    if (!valid_sizes(nx, ny, nz)) return fail(ARK_EINVAL, "ark_create: need nx,ny >= 4 and nz == 1 or nz >= 4%s");
    if (!(dx > 0.0) || !(gamma > 1.0) || !(mu >= 0.0) || !(kappa >= 0.0) || !g || !bc)
        return fail(ARK_EINVAL, "ark_create: need dx > 0, gamma > 1, mu,kappa >= 0, g and bc non-NULL%s");
    if (low_mach_theta != 0 && low_mach_theta != 1) return fail(ARK_EINVAL, "ark_create: low_mach_theta must be 0 or 1%s");
    const int ndim = nz > 1 ? 3 : 2;
    for (int d = 0; d < ndim; ++d) {
        for (int sd = 0; sd < 2; ++sd) {
            const int t = bc->type[d][sd];
            if (t != ARK_BC_PERIODIC && t != ARK_BC_REFLECTING && t != ARK_BC_FIXED_T_WALL && t != ARK_BC_FLUX_WALL && t != ARK_BC_EXTERNAL)
                return fail(ARK_EINVAL, "ark_create: unknown boundary kind%s");
            if (t == ARK_BC_EXTERNAL && !(ndim == 3 && d == 2))
                return fail(ARK_EINVAL, "ark_create: ARK_BC_EXTERNAL (slab decomposition) exists on the z axis of 3D grids only%s");
            if (t == ARK_BC_FLUX_WALL && !(kappa > 0.0))
                return fail(ARK_EINVAL, "ark_create: an imposed-flux wall needs kappa > 0%s");
            if (t == ARK_BC_FIXED_T_WALL && !(bc->value[d][sd] > 0.0))
                return fail(ARK_EINVAL, "ark_create: fixed-T wall needs a positive temperature%s");
        }
        if ((bc->type[d][0] == ARK_BC_PERIODIC) != (bc->type[d][1] == ARK_BC_PERIODIC))
            return fail(ARK_EINVAL, "ark_create: periodic must be set on both sides of an axis%s");
    }
    const Layout L = make_layout(nx, ny, nz);
    if (!d_workspace || workspace_bytes < L.total || ((size_t)d_workspace & 255))
        return fail(ARK_EINVAL, "ark_create: workspace NULL, misaligned (256 B) or smaller than ark_workspace_bytes()%s");

    {   // the handle lives on the CURRENT device (kernel attributes, launches): its workspace must be memory of that device
        int dev = -1;
        cudaPointerAttributes at;
        ARK_CUDA(cudaGetDevice(&dev));
        ARK_CUDA(cudaPointerGetAttributes(&at, d_workspace));
        if ((at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) || (at.type == cudaMemoryTypeDevice && at.device != dev))
            return fail(ARK_EINVAL, "ark_create: the workspace is not device memory of the current CUDA device (%s%lld); make the "
                                    "workspace's device current before calling", "", (long long)dev);
    }
    ark_solver* s = new (std::nothrow) ark_solver;
    if (!s) return fail(ARK_ENOMEM, "ark_create: out of host memory%s");
    memset(s, 0, sizeof *s);
    ArkParams& P = s->P;
    P.nx = nx; P.ny = ny; P.nz = nz; P.ndim = ndim; P.nf = L.nf;
    P.px = L.px; P.py = L.py; P.pz = L.pz; P.offz = L.offz; P.fstride = L.fstride;
    P.h = dx; P.gamma = gamma; P.gm1 = gamma - 1.0; P.mu = mu; P.kappa = kappa; P.theta = low_mach_theta;
    for (int d = 0; d < 3; ++d) {
        P.g[d] = d < ndim ? g[d] : 0.0;
        for (int sd = 0; sd < 2; ++sd) { P.bc[d][sd] = bc->type[d][sd]; P.bcv[d][sd] = bc->value[d][sd]; }
    }
    ark_fill_derived(P);
    s->L = L;
    s->ws = (char*)d_workspace;
    s->U[0] = (double*)s->ws;
    s->U[1] = (double*)(s->ws + L.state_bytes);
    s->cur = 0;
    s->scratch = (double*)(s->ws + L.scratch_off);
    s->result = (double*)(s->ws + L.result_off);
    s->dtlog = (double*)(s->ws + L.dtlog_off);
    s->stage = (double*)(s->ws + L.stage_off);
    s->stream = (cudaStream_t)cuda_stream;
    s->rate_slots = 0;
    s->launches = 0;
    { cudaError_t e0 = cudaGetDevice(&s->device); if (e0 != cudaSuccess) { delete s; return fail(ARK_ECUDA, "CUDA error: %s", cudaGetErrorString(e0)); } }

    // launch geometry of the fused step kernel
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, s->device);
    if (nsm < 1) nsm = 148;
    s->zchunk = 0;                                              // the kernel reads the chunk table P.zb
    if (step_blocks(nx, ny, nz, &s->step_grid, s->P.zb, nsm) > MAX_SCRATCH - DIAG_BLOCKS * ARK_NDIAG) {
        delete s;
        return fail(ARK_EINVAL, "ark_create: grid too large for the per-block rate scratch (ark_workspace_bytes returns 0 for it)%s");
    }
    if (ndim == 3) {
        for (int b = 0; b < 2; ++b) {
            const int rc = make_tensor_map(&s->tmap[b], L, s->U[b], TX3 + 4, TY3 + 4);
            if (rc != ARK_OK) { delete s; return rc; }
        }
    }
    { const int rc = set_step_attributes(ndim); if (rc != ARK_OK) { delete s; return rc; } }
    cudaError_t e = cudaMallocHost((void**)&s->h_pinned, 2 * sizeof(double));
    if (e != cudaSuccess) { delete s; return fail(ARK_ECUDA, "CUDA error: %s", cudaGetErrorString(e)); }
    // ghost cells and padding start finite (they are read by clamped / halo threads before the first fill)
    e = cudaMemsetAsync(s->ws, 0, L.total, s->stream);
    if (e != cudaSuccess) { cudaFreeHost(s->h_pinned); delete s; return fail(ARK_ECUDA, "CUDA error: %s", cudaGetErrorString(e)); }
    *out = s;
    return ARK_OK;
}

int ark_step_kernel_timing(ark_solver* s, int enable) {
    if (!s) return fail(ARK_EINVAL, "ark_step_kernel_timing: NULL handle%s");
    if (enable && !s->timer) {
        s->timer = new (std::nothrow) ArkTimer;
        if (!s->timer) return fail(ARK_ENOMEM, "ark_step_kernel_timing: out of host memory%s");
        for (int i = 0; i < ARK_MAX_TIMED; ++i) {
            ARK_CUDA(cudaEventCreate(&s->timer->ev0[i]));
            ARK_CUDA(cudaEventCreate(&s->timer->ev1[i]));
        }
    }
    s->timing = enable != 0;
    s->n_timed = 0;
    return ARK_OK;
}

int ark_step_kernel_time(ark_solver* s, double* total_ms, int* launches) {
    if (!s || !total_ms || !launches) return fail(ARK_EINVAL, "ark_step_kernel_time: NULL argument%s");
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    double sum = 0.0;
    for (int i = 0; i < s->n_timed; ++i) {
        float ms = 0.f;
        ARK_CUDA(cudaEventElapsedTime(&ms, s->timer->ev0[i], s->timer->ev1[i]));
        sum += ms;
    }
    *total_ms = sum;
    *launches = s->n_timed;
    return ARK_OK;
}

void ark_destroy(ark_solver* s) {
    if (!s) return;
    if (s->timer) {
        for (int i = 0; i < ARK_MAX_TIMED; ++i) { cudaEventDestroy(s->timer->ev0[i]); cudaEventDestroy(s->timer->ev1[i]); }
        delete s->timer;
    }
    if (s->h_pinned) cudaFreeHost(s->h_pinned);
    if (s->gexec) cudaGraphExecDestroy(s->gexec);
    if (s->gstream) { cudaEventDestroy(s->gev_in); cudaEventDestroy(s->gev_out); cudaStreamDestroy(s->gstream); }
    delete s;
}

long long ark_launch_count(const ark_solver* s) { return s ? s->launches : 0; }

int ark_set_state(ark_solver* s, const double* rho, const double* rhou, const double* rhov, const double* rhow,
                  const double* E) {
    if (!s || !rho || !rhou || !rhov || !E || (s->P.ndim == 3 && !rhow)) return fail(ARK_EINVAL, "ark_set_state: NULL argument%s");
    ARK_ON_DEVICE(s);
    const double* src[5] = {rho, rhou, rhov, s->P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
    for (int f = 0; f < s->P.nf; ++f) {
        ark_k_pack<<<grid_for(n, 256), 256, 0, s->stream>>>(s->P, s->U[s->cur], (s->P.ndim == 3 || f < 3) ? src[f] : E, f);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    s->rate_slots = 0;
    s->xghost_valid = false;
    s->yghost_valid = false;
    s->xyghost_valid = false;
    return ARK_OK;
}

int ark_get_state(ark_solver* s, double* rho, double* rhou, double* rhov, double* rhow, double* E) {
    if (!s || !rho || !rhou || !rhov || !E || (s->P.ndim == 3 && !rhow)) return fail(ARK_EINVAL, "ark_get_state: NULL argument%s");
    ARK_ON_DEVICE(s);
    double* dst[5] = {rho, rhou, rhov, s->P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
    for (int f = 0; f < s->P.nf; ++f) {
        ark_k_unpack<<<grid_for(n, 256), 256, 0, s->stream>>>(s->P, s->U[s->cur], (s->P.ndim == 3 || f < 3) ? dst[f] : E, f);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

int ark_set_state_host(ark_solver* s, const double* rho, const double* rhou, const double* rhov, const double* rhow,
                       const double* E) {
    if (!s || !rho || !rhou || !rhov || !E || (s->P.ndim == 3 && !rhow)) return fail(ARK_EINVAL, "ark_set_state_host: NULL argument%s");
    ARK_ON_DEVICE(s);
    const double* src[5] = {rho, rhou, rhov, s->P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
    for (int f = 0; f < s->P.nf; ++f) {
        const double* h = (s->P.ndim == 3 || f < 3) ? src[f] : E;
        ARK_CUDA(cudaMemcpyAsync(s->stage, h, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, s->stream));
        ark_k_pack<<<grid_for(n, 256), 256, 0, s->stream>>>(s->P, s->U[s->cur], s->stage, f);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    s->rate_slots = 0;
    s->xghost_valid = false;
    s->yghost_valid = false;
    s->xyghost_valid = false;
    return ARK_OK;
}

int ark_get_state_host(ark_solver* s, double* rho, double* rhou, double* rhov, double* rhow, double* E) {
    if (!s || !rho || !rhou || !rhov || !E || (s->P.ndim == 3 && !rhow)) return fail(ARK_EINVAL, "ark_get_state_host: NULL argument%s");
    ARK_ON_DEVICE(s);
    double* dst[5] = {rho, rhou, rhov, s->P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
    for (int f = 0; f < s->P.nf; ++f) {
        double* h = (s->P.ndim == 3 || f < 3) ? dst[f] : E;
        ark_k_unpack<<<grid_for(n, 256), 256, 0, s->stream>>>(s->P, s->U[s->cur], s->stage, f);
        s->launches++;
        ARK_CUDA(cudaMemcpyAsync(h, s->stage, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    }
    ARK_CUDA(cudaGetLastError());
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    return ARK_OK;
}

int ark_compute_dt(ark_solver* s, double cfl, double* dt_out) {
    if (!s || !dt_out || !(cfl > 0.0)) return fail(ARK_EINVAL, "ark_compute_dt: bad argument%s");
    ARK_ON_DEVICE(s);
    int rc = reduce_rate(s, cfl, nullptr);
    if (rc != ARK_OK) return rc;
    ARK_CUDA(cudaMemcpyAsync(s->h_pinned, s->result, 2 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    const double rate = s->h_pinned[0];
    if (!(rate > 0.0) || std::isinf(rate) || std::isnan(rate)) {
        *dt_out = std::nan("");
        return fail(ARK_ENONFINITE, "ark_compute_dt: maximum CFL rate is not finite and positive%s");
    }
    *dt_out = cfl / rate;
    return ARK_OK;
}

int ark_step(ark_solver* s, double dt) {
    if (!s || !(dt > 0.0) || std::isinf(dt)) return fail(ARK_EINVAL, "ark_step: dt must be finite and positive%s");
    ARK_ON_DEVICE(s);
    return do_step(s, dt, nullptr);
}

// Device-side halves of {ark_compute_dt; ark_step} for time loops that must not wait for the host (see ark.h)
int ark_max_rate_device(ark_solver* s, double* d_rate_out) {
    if (!s || !d_rate_out) return fail(ARK_EINVAL, "ark_max_rate_device: NULL argument%s");
    ARK_ON_DEVICE(s);
    const int rc = reduce_rate(s, 1.0, nullptr);                 // result[0] = max rate of the current state
    if (rc != ARK_OK) return rc;
    ARK_CUDA(cudaMemcpyAsync(d_rate_out, s->result, sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return ARK_OK;
}

int ark_step_device_dt(ark_solver* s, const double* d_dt) {
    if (!s || !d_dt) return fail(ARK_EINVAL, "ark_step_device_dt: NULL argument%s");
    ARK_ON_DEVICE(s);
    // the step kernels read a device-side step size from result[1] (where pass 2 of ark_run leaves it)
    ARK_CUDA(cudaMemcpyAsync(s->result + 1, d_dt, sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return do_step(s, 0.0, s->result);
}

namespace {

// one step of the device-side loop: dt = cfl / max rate (pass 2 on the rates of the current state), then the step
int run_one(ark_solver* s, double cfl, double* dt_log) {
    int rc = reduce_rate(s, cfl, dt_log);
    if (rc != ARK_OK) return rc;
    return do_step(s, 0.0, s->result);
}

// npairs x (two steps) replayed from a CUDA graph captured on the library's own stream; the caller's stream waits
// for it through events.  The graph is cached and re-captured when the buffer parity, cfl or logging changes.
int run_pairs_graph(ark_solver* s, int npairs, double cfl, double* dt_log) {
    if (!s->gstream) {
        ARK_CUDA(cudaStreamCreateWithFlags(&s->gstream, cudaStreamNonBlocking));
        ARK_CUDA(cudaEventCreateWithFlags(&s->gev_in, cudaEventDisableTiming));
        ARK_CUDA(cudaEventCreateWithFlags(&s->gev_out, cudaEventDisableTiming));
    }
    if (!s->gexec || s->g_cur != s->cur || s->g_cfl != cfl || s->g_log != (dt_log != nullptr)) {
        if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
        const cudaStream_t user = s->stream;
        const long long l0 = s->launches;
        s->stream = s->gstream;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamBeginCapture(s->gstream, cudaStreamCaptureModeThreadLocal);
        int rc = e == cudaSuccess ? ARK_OK : fail(ARK_ECUDA, "CUDA error: %s (graph capture)", cudaGetErrorString(e));
        if (rc == ARK_OK) rc = run_one(s, cfl, dt_log);
        if (rc == ARK_OK) rc = run_one(s, cfl, dt_log);
        if (e == cudaSuccess) {
            const cudaError_t e2 = cudaStreamEndCapture(s->gstream, &graph);
            if (rc == ARK_OK && e2 != cudaSuccess) rc = fail(ARK_ECUDA, "CUDA error: %s (graph capture)", cudaGetErrorString(e2));
        }
        s->stream = user;
        s->g_launches = s->launches - l0;
        s->launches = l0;                       // nothing ran yet; (cur flipped twice: unchanged)
        if (rc == ARK_OK) {
            const cudaError_t e3 = cudaGraphInstantiate(&s->gexec, graph, 0);
            if (e3 != cudaSuccess) rc = fail(ARK_ECUDA, "CUDA error: %s (graph instantiate)", cudaGetErrorString(e3));
        }
        if (graph) cudaGraphDestroy(graph);
        if (rc != ARK_OK) { s->gexec = nullptr; return rc; }
        s->g_cur = s->cur; s->g_cfl = cfl; s->g_log = dt_log != nullptr;
    }
    ARK_CUDA(cudaEventRecord(s->gev_in, s->stream));
    ARK_CUDA(cudaStreamWaitEvent(s->gstream, s->gev_in, 0));
    for (int i = 0; i < npairs; ++i) ARK_CUDA(cudaGraphLaunch(s->gexec, s->gstream));
    ARK_CUDA(cudaEventRecord(s->gev_out, s->gstream));
    ARK_CUDA(cudaStreamWaitEvent(s->stream, s->gev_out, 0));
    s->launches += s->g_launches * npairs;
    return ARK_OK;
}

}  // namespace

int ark_run(ark_solver* s, int nsteps, double cfl, double* dts_out) {
    if (!s || nsteps < 0 || !(cfl > 0.0)) return fail(ARK_EINVAL, "ark_run: bad argument%s");
    ARK_ON_DEVICE(s);
    if (s->P.ndim == 3 && (s->P.bc[2][0] == ARK_BCK_EXTERNAL || s->P.bc[2][1] == ARK_BCK_EXTERNAL))
        return fail(ARK_EINVAL, "ark_run: a sub-domain with external ghost planes needs a halo exchange before every step%s");
    if (dts_out && nsteps > DTLOG_MAX) return fail(ARK_EINVAL, "ark_run: at most %s%lld steps when dts_out is given", "", (long long)DTLOG_MAX);
    double* dt_log = dts_out ? s->dtlog : nullptr;
    // result[3]: sticky "a rate was not finite and positive" flag of pass 2; result[4]: log counter
    ARK_CUDA(cudaMemsetAsync(s->result + 3, 0, 2 * sizeof(double), s->stream));
    int done = 0;
    // the first step may need the standalone rate pass; from then on every step has the same launch sequence
    if (nsteps > 0) { const int rc = run_one(s, cfl, dt_log); if (rc != ARK_OK) return rc; done = 1; }
    if (!s->timing && nsteps - done >= 4) {
        const int npairs = (nsteps - done) / 2;
        const int rc = run_pairs_graph(s, npairs, cfl, dt_log);
        if (rc != ARK_OK) return rc;
        done += 2 * npairs;
    }
    for (; done < nsteps; ++done) { const int rc = run_one(s, cfl, dt_log); if (rc != ARK_OK) return rc; }
    if (nsteps > 0) {
        // one synchronisation per call: the non-finite flag (and the step sizes if asked for)
        if (dts_out) ARK_CUDA(cudaMemcpyAsync(dts_out, s->dtlog, (size_t)nsteps * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        ARK_CUDA(cudaMemcpyAsync(s->h_pinned, s->result + 3, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        ARK_CUDA(cudaStreamSynchronize(s->stream));
        if (s->h_pinned[0] != 0.0) return fail(ARK_ENONFINITE, "ark_run: a maximum CFL rate was not finite and positive%s");
    }
    return ARK_OK;
}

int ark_diagnostics(ark_solver* s, double* out) {
    if (!s || !out) return fail(ARK_EINVAL, "ark_diagnostics: NULL argument%s");
    ARK_ON_DEVICE(s);
    const long long n = (long long)s->P.nx * s->P.ny * s->P.nz;
    const int nb = grid_for(n, 256, DIAG_BLOCKS);
    double* part = s->scratch + (MAX_SCRATCH - DIAG_BLOCKS * ARK_NDIAG);     // tail of the rate scratch (see ark_create)
    double* res = s->result + 8;
    ark_k_diag_pass1<<<nb, 256, 0, s->stream>>>(s->P, s->U[s->cur], part);
    ark_k_diag_pass2<<<1, 256, 0, s->stream>>>(part, nb, res);
    s->launches += 2;
    ARK_CUDA(cudaGetLastError());
    double h[ARK_NDIAG];
    ARK_CUDA(cudaMemcpyAsync(h, res, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    double vol = 1.0;
    for (int d = 0; d < s->P.ndim; ++d) vol *= s->P.h;
    out[0] = h[0];                 // max |u|
    out[1] = h[1] / (double)n;     // mean |u|
    out[2] = h[2] * vol;           // kinetic energy
    out[3] = h[3];                 // max Mach number
    out[4] = h[4] * vol;           // mass
    out[5] = h[5] * vol;           // total energy incl. potential
    return ARK_OK;
}

int ark_set_energy_form(ark_solver* s, int form) {
    if (!s || (form != ARK_ENERGY_CONSERVATIVE && form != ARK_ENERGY_APPENDIX_B)) return fail(ARK_EINVAL, "ark_set_energy_form: form must be 0 or 1%s");
    s->P.eform = form;
    if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }   // the captured launches carry the old parameters
    return ARK_OK;
}

size_t ark_potential_bytes(int nx, int ny, int nz) {
    if (!supported_grid(nx, ny, nz)) return 0;
    return (size_t)make_layout(nx, ny, nz).fstride * sizeof(double);
}

int ark_set_potential(ark_solver* s, const double* d_phi, void* d_buffer, size_t buffer_bytes) {
    if (!s) return fail(ARK_EINVAL, "ark_set_potential: NULL handle%s");
    ARK_ON_DEVICE(s);
    ArkParams& P = s->P;
    if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
    // wall ghost cells carry the hydrostatic extrapolation for the potential that was set when they were filled
    // (relation (14) with the potential difference): whatever sweeps already ran on the current state are stale now
    s->xghost_valid = s->yghost_valid = s->xyghost_valid = false;
    if (d_phi && P.ndim == 3 && (P.bc[2][0] == ARK_BCK_EXTERNAL || P.bc[2][1] == ARK_BCK_EXTERNAL))
        return fail(ARK_EINVAL, "ark_set_potential: not available on a sub-domain with external ghost planes%s");
    if (!d_phi) {                                   // back to the constant gravity vector of ark_create
        P.phi = nullptr;
        ark_fill_derived(P);
        return ARK_OK;
    }
    const size_t need = (size_t)P.fstride * sizeof(double);
    if (!d_buffer || buffer_bytes < need || ((size_t)d_buffer & 255))
        return fail(ARK_EINVAL, "ark_set_potential: buffer NULL, misaligned (256 B) or smaller than ark_potential_bytes()%s");
    double* pad = (double*)d_buffer;
    ARK_CUDA(cudaMemsetAsync(pad, 0, need, s->stream));
    const long long n = (long long)P.nx * P.ny * P.nz;
    ark_k_pack<<<grid_for(n, 256), 256, 0, s->stream>>>(P, pad, d_phi, 0);
    ark_k_phi_ghosts<0><<<grid_for((long long)P.ny * P.nz, 128), 128, 0, s->stream>>>(P, pad);
    ark_k_phi_ghosts<1><<<grid_for((long long)(P.nx + 2 * ARK_NG) * P.nz, 128), 128, 0, s->stream>>>(P, pad);
    s->launches += 3;
    if (P.ndim == 3) {
        ark_k_phi_ghosts<2><<<grid_for((long long)(P.nx + 2 * ARK_NG) * (P.ny + 2 * ARK_NG), 128), 128, 0, s->stream>>>(P, pad);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    P.phi = pad;
    for (int d = 0; d < P.ndim; ++d) P.D.g_on[d] = 1;          // every axis carries gravity terms now
    return ARK_OK;
}

size_t ark_halo_bytes(int nx, int ny, int nz) {
    if (!supported_grid(nx, ny, nz) || nz == 1) return 0;
    const Layout L = make_layout(nx, ny, nz);
    return (size_t)L.nf * ARK_NG * L.px * L.py * sizeof(double);
}

int ark_get_halo(ark_solver* s, int side, double* d_buf) {
    if (!s || !d_buf || (side != 0 && side != 1) || s->P.ndim != 3) return fail(ARK_EINVAL, "ark_get_halo: bad argument (3D solvers only)%s");
    ARK_ON_DEVICE(s);
    // the planes travel with their x / y ghost cells: those sweeps run now (and are skipped by the next ark_step)
    const int rc = launch_bc_xy(s, s->U[s->cur]);
    if (rc != ARK_OK) return rc;
    s->xyghost_valid = true;
    const ArkParams& P = s->P;
    const size_t plane = (size_t)P.px * P.py, chunk = ARK_NG * plane;
    const int k0 = side == 0 ? 0 : P.nz - ARK_NG;                    // the two interior planes next to that side
    for (int f = 0; f < P.nf; ++f)
        ARK_CUDA(cudaMemcpyAsync(d_buf + f * chunk, s->U[s->cur] + f * P.fstride + (size_t)(k0 + P.offz) * plane, chunk * sizeof(double),
                                 cudaMemcpyDeviceToDevice, s->stream));
    return ARK_OK;
}

int ark_set_halo(ark_solver* s, int side, const double* d_buf) {
    if (!s || !d_buf || (side != 0 && side != 1) || s->P.ndim != 3) return fail(ARK_EINVAL, "ark_set_halo: bad argument (3D solvers only)%s");
    ARK_ON_DEVICE(s);
    if (s->P.bc[2][side] != ARK_BCK_EXTERNAL) return fail(ARK_EINVAL, "ark_set_halo: that side is not ARK_BC_EXTERNAL%s");
    const ArkParams& P = s->P;
    const size_t plane = (size_t)P.px * P.py, chunk = ARK_NG * plane;
    const int k0 = side == 0 ? -ARK_NG : P.nz;                       // the two ghost planes of that side
    for (int f = 0; f < P.nf; ++f)
        ARK_CUDA(cudaMemcpyAsync(s->U[s->cur] + f * P.fstride + (size_t)(k0 + P.offz) * plane, d_buf + f * chunk, chunk * sizeof(double),
                                 cudaMemcpyDeviceToDevice, s->stream));
    return ARK_OK;
}

int ark_ke_spectrum_bins(int nx, int ny) {
    if (nx < 4 || ny < 4) return 0;
    return (int)std::floor(std::sqrt((double)(nx / 2) * (nx / 2) + (double)(ny / 2) * (ny / 2)) + 0.5) + 1;
}

int ark_ke_spectrum(ark_solver* s, double* out, int nbins) {
    if (!s || !out) return fail(ARK_EINVAL, "ark_ke_spectrum: NULL argument%s");
    ARK_ON_DEVICE(s);
    const ArkParams& P = s->P;
    if (P.ndim != 3 || P.nz < 8) return fail(ARK_EINVAL, "ark_ke_spectrum: needs a 3D grid with nz >= 8 (scratch lives in the staging field)%s");
    if (nbins != ark_ke_spectrum_bins(P.nx, P.ny) || nbins > 4096) return fail(ARK_EINVAL, "ark_ke_spectrum: nbins must be ark_ke_spectrum_bins(nx, ny)%s");
    // scratch inside the dense staging field (nx*ny*nz doubles): A 6 nx ny | Pw nx ny | twiddles 2 nx + 2 ny | E nbins
    const long long n = (long long)P.nx * P.ny;
    if (7 * n + 2 * (P.nx + P.ny) + nbins > n * P.nz) return fail(ARK_EINVAL, "ark_ke_spectrum: grid too thin for the scratch%s");
    double* A = s->stage;
    double* Pw = A + 6 * n;
    double* twx = Pw + n;
    double* twy = twx + 2 * P.nx;
    double* E = twy + 2 * P.ny;
    ark_k_spec_twiddle<<<grid_for(P.nx, 128), 128, 0, s->stream>>>(twx, P.nx);
    ark_k_spec_twiddle<<<grid_for(P.ny, 128), 128, 0, s->stream>>>(twy, P.ny);
    ark_k_spec_rows<<<grid_for(n, 128, 148 * 16), 128, 0, s->stream>>>(P, s->U[s->cur], P.nz / 2, twx, A);
    ark_k_spec_cols<<<grid_for(n, 128, 148 * 16), 128, 0, s->stream>>>(P, A, twy, Pw);
    ark_k_spec_bins<<<nbins, 256, 0, s->stream>>>(P, Pw, E);
    s->launches += 5;
    ARK_CUDA(cudaGetLastError());
    ARK_CUDA(cudaMemcpyAsync(out, E, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    ARK_CUDA(cudaStreamSynchronize(s->stream));
    return ARK_OK;
}

int ark_measure_fp64_peak(double* tinstr_per_s, void* cuda_stream) {
    if (!tinstr_per_s) return fail(ARK_EINVAL, "ark_measure_fp64_peak: NULL argument%s");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    ARK_CUDA(cudaGetDevice(&dev));
    ARK_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    ARK_CUDA(cudaMalloc((void**)&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    ARK_CUDA(cudaEventCreate(&e0));
    ARK_CUDA(cudaEventCreate(&e1));
    const int threads = 512, blocks = nsm * 2, iters = 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {          // the first repetition warms up
        ARK_CUDA(cudaEventRecord(e0, st));
        ark_k_dfma_peak<<<blocks, threads, 0, st>>>(sink, iters, 0.999999, 1e-7);
        ARK_CUDA(cudaEventRecord(e1, st));
        ARK_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        ARK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double rate = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3) / 1e12;
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    ARK_CUDA(cudaGetLastError());
    *tinstr_per_s = best;
    return ARK_OK;
}

int ark_debug_get_padded(ark_solver* s, double* rho, double* rhou, double* rhov, double* rhow, double* E) {
    if (!s || !rho || !rhou || !rhov || !E || (s->P.ndim == 3 && !rhow)) return fail(ARK_EINVAL, "ark_debug_get_padded: NULL argument%s");
    ARK_ON_DEVICE(s);
    int rc = launch_bc(s, s->U[s->cur]);
    if (rc != ARK_OK) return rc;
    double* dst[5] = {rho, rhou, rhov, s->P.ndim == 3 ? rhow : E, E};
    const long long n = (long long)(s->P.nx + 2 * ARK_NG) * s->P.py * s->P.pz;
    for (int f = 0; f < s->P.nf; ++f) {
        ark_k_unpack_padded<<<grid_for(n, 256), 256, 0, s->stream>>>(s->P, s->U[s->cur], (s->P.ndim == 3 || f < 3) ? dst[f] : E, f);
        s->launches++;
    }
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// ark_cfl_dt_static: the CFL time step without any device allocation (see include/ark.h for who needs that and why).
//
// The two-pass max reduction needs one double of scratch per block of pass 1.  Every other entry point takes that
// scratch from the caller's workspace; this one keeps it in the library image: a file-scope device array of
// ARK_STATIC_SLOTS doubles (256 KiB) that every GPU which loads the library holds until the process exits.  Pass 1 is a
// variant of ark_k_cfl_pass1 that reads the caller's DENSE fields directly (no padded copy, so no second buffer either)
// and gives every block a fixed range of ARK_STATIC_BLOCK_CELLS cells, which is what bounds the grid size: at most
// ARK_STATIC_SLOTS * ARK_STATIC_BLOCK_CELLS = 2^27 cells (512^3).
//
// In host code `g_static_rates` is only the host-side shadow of the symbol, not a device address; the address the kernels
// get comes from cudaGetSymbolAddress, asked for once per device while that device is current (static_rates_ptr below).
// ------------------------------------------------------------------------------------------------
#define ARK_STATIC_SLOTS 32768
#define ARK_STATIC_BLOCK_THREADS 256
#define ARK_STATIC_CELLS_PER_THREAD 16
#define ARK_STATIC_BLOCK_CELLS (ARK_STATIC_BLOCK_THREADS * ARK_STATIC_CELLS_PER_THREAD)
#define ARK_STATIC_MAX_DEVICES 64

static __device__ __align__(256) double g_static_rates[ARK_STATIC_SLOTS];

// pass 1 on dense fields: block b owns cells [b * BLOCK_CELLS, (b + 1) * BLOCK_CELLS), coalesced strides of one block
// width; slots[b] = NaN-propagating max of the cells' CFL rates.  Every slot a call reads is written by that call first.
static __global__ void __launch_bounds__(ARK_STATIC_BLOCK_THREADS)
ark_k_cfl_dense_pass1(ArkParams P, long long n, const double* __restrict__ rho, const double* __restrict__ mx,
                      const double* __restrict__ my, const double* __restrict__ mz, const double* __restrict__ E,
                      double* __restrict__ slots) {
    __shared__ double red[32];
    const double inv_h = 1.0 / P.h;
    const double dcoef = 2.0 * P.ndim * fmax(4.0 * P.mu / 3.0, P.gm1 * P.kappa) * inv_h * inv_h;
    const long long base = (long long)blockIdx.x * ARK_STATIC_BLOCK_CELLS + threadIdx.x;
    double m = -1.0;
#pragma unroll 4
    for (int j = 0; j < ARK_STATIC_CELLS_PER_THREAD; ++j) {
        const long long c = base + (long long)j * ARK_STATIC_BLOCK_THREADS;
        if (c < n) m = ark_nanmax(m, ark_rate(P, rho[c], mx[c], my[c], P.ndim == 3 ? mz[c] : 0.0, E[c], inv_h, dcoef));
    }
    m = ark_block_nanmax(m, red);
    if (threadIdx.x == 0) slots[blockIdx.x] = m;
}

// pass 2: one block over the nvals slots of this call; out[0] = max rate, out[1] = cfl / max rate
static __global__ void ark_k_cfl_static_pass2(const double* __restrict__ slots, int nvals, double cfl, double* __restrict__ out) {
    __shared__ double red[32];
    double m = -1.0;
    for (int s = threadIdx.x; s < nvals; s += blockDim.x) m = ark_nanmax(m, slots[s]);
    m = ark_block_nanmax(m, red);
    if (threadIdx.x == 0) { out[0] = m; out[1] = cfl / m; }
}

namespace {

// Device address of g_static_rates on the CURRENT device, looked up once per device ordinal.  (The runtime resolves the
// symbol against the current device's copy of the module, so the look-up must happen with that device current; the
// result is a plain device pointer that stays valid until the process exits.)
int static_rates_ptr(double** out) {
    static double* cached[ARK_STATIC_MAX_DEVICES];     // zero-initialised; written once per device
    int dev = -1;
    ARK_CUDA(cudaGetDevice(&dev));
    const bool slot = dev >= 0 && dev < ARK_STATIC_MAX_DEVICES;
    double* p = slot ? __atomic_load_n(&cached[dev], __ATOMIC_ACQUIRE) : nullptr;
    if (!p) {
        void* q = nullptr;
        ARK_CUDA(cudaGetSymbolAddress(&q, g_static_rates));
        if (!q) return fail(ARK_ECUDA, "ark_cfl_dt_static: cudaGetSymbolAddress returned no address%s");
        p = (double*)q;
        if (slot) __atomic_store_n(&cached[dev], p, __ATOMIC_RELEASE);   // two racing threads store the same value
    }
    *out = p;
    return ARK_OK;
}

}  // namespace

extern "C" {

size_t ark_cfl_dt_static_max_cells(void) { return (size_t)ARK_STATIC_SLOTS * ARK_STATIC_BLOCK_CELLS; }

int ark_cfl_dt_static(int nx, int ny, int nz, double dx, double gamma, double mu, double kappa, const double* rho,
                      const double* rhou, const double* rhov, const double* rhow, const double* E, double cfl,
                      double* d_out, void* cuda_stream) {
    if (!valid_sizes(nx, ny, nz)) return fail(ARK_EINVAL, "ark_cfl_dt_static: need nx,ny >= 4 and nz == 1 or nz >= 4, each <= 16384%s");
    if (!(dx > 0.0) || !(gamma > 1.0) || !(mu >= 0.0) || !(kappa >= 0.0) || !(cfl > 0.0))
        return fail(ARK_EINVAL, "ark_cfl_dt_static: need dx > 0, gamma > 1, mu,kappa >= 0, cfl > 0%s");
    if (!rho || !rhou || !rhov || !E || (nz > 1 && !rhow) || !d_out) return fail(ARK_EINVAL, "ark_cfl_dt_static: NULL argument%s");
    const long long n = (long long)nx * ny * nz;
    if (n > (long long)ark_cfl_dt_static_max_cells())
        return fail(ARK_EINVAL, "ark_cfl_dt_static: the grid has more cells than the library's built-in scratch serves%s (at most %lld = 512^3; "
                                "larger grids: ark_compute_dt with a caller-allocated workspace)", "", (long long)ark_cfl_dt_static_max_cells());
    double* slots = nullptr;
    { const int rc = static_rates_ptr(&slots); if (rc != ARK_OK) return rc; }
    ArkParams P;
    memset(&P, 0, sizeof P);
    P.nx = nx; P.ny = ny; P.nz = nz; P.ndim = nz > 1 ? 3 : 2;
    P.h = dx; P.gamma = gamma; P.gm1 = gamma - 1.0; P.mu = mu; P.kappa = kappa;
    const int nblocks = (int)((n + ARK_STATIC_BLOCK_CELLS - 1) / ARK_STATIC_BLOCK_CELLS);
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    ark_k_cfl_dense_pass1<<<nblocks, ARK_STATIC_BLOCK_THREADS, 0, st>>>(P, n, rho, rhou, rhov, rhow, E, slots);
    ark_k_cfl_static_pass2<<<1, 1024, 0, st>>>(slots, nblocks, cfl, d_out);
    ARK_CUDA(cudaGetLastError());
    return ARK_OK;
}

}  // extern "C"
