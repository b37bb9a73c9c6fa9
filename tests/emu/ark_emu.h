// ark_emu.h -- TEST-ONLY host emulation shim for the CUDA kernel headers (paper_1903_09043_b200/csrc/*.cuh).
// With -DARK_HOST_EMU the kernels compile as plain C++: one std::thread per CUDA thread of a block, blocks run
// one after another, __syncthreads() is a std::barrier.  It lets `pytest -m "not gpu"` exercise the kernels'
// indexing, tiling, halo and pipeline logic on a CPU-only box (tests/test_emu_kernels.py).  It is never part of
// the product library (libark_b200.so is built by nvcc only) and is not a fallback.
#pragma once
#include <algorithm>
#include <barrier>
#include <cmath>
#include <cstring>
#include <functional>
#include <memory>
#include <thread>
#include <vector>

struct emu_dim3 { unsigned x = 1, y = 1, z = 1; };
inline thread_local emu_dim3 threadIdx, blockIdx, blockDim, gridDim;
inline double* ark_emu_smem = nullptr;
inline std::barrier<>* ark_emu_barrier = nullptr;
inline std::vector<double> ark_emu_red;

#define ARK_DEV inline
#define ARK_GLOBAL inline
#define ARK_SHARED static
#define ARK_DYN_SMEM(name) double* name = ark_emu_smem
#define __syncthreads() ark_emu_barrier->arrive_and_wait()

inline double rsqrt(double x) { return 1.0 / std::sqrt(x); }
inline long long __double_as_longlong(double x) { long long r; std::memcpy(&r, &x, 8); return r; }
inline double __longlong_as_double(long long x) { double r; std::memcpy(&r, &x, 8); return r; }

inline double ark_emu_block_nanmax(double v) {
    ark_emu_red[threadIdx.x] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (unsigned i = 1; i < blockDim.x; ++i) {
            const double b = ark_emu_red[i];
            v = (v != v) ? v : ((b != b) ? b : (v > b ? v : b));
        }
    }
    __syncthreads();
    return v;
}

// Warp shuffles (3D step kernel: x-neighbour exchange).  A "warp" of the emulation is ark_emu_warp consecutive
// threads of the block (the kernel's region width); every thread of a warp calls the same shuffle sequence, so a
// per-warp barrier on both sides of a small exchange array reproduces __shfl_up/down_sync(.., 1).
inline unsigned ark_emu_warp = 32;
inline std::vector<std::unique_ptr<std::barrier<>>> ark_emu_wbar;
inline std::vector<double> ark_emu_shfl_buf;
inline double ark_emu_shfl(double v, int delta) {
    const unsigned t = threadIdx.x, w = t / ark_emu_warp, lane = t % ark_emu_warp;
    ark_emu_shfl_buf[t] = v;
    ark_emu_wbar[w]->arrive_and_wait();
    const int src = (int)lane + delta;
    const double r = (src >= 0 && src < (int)ark_emu_warp) ? ark_emu_shfl_buf[w * ark_emu_warp + src] : v;
    ark_emu_wbar[w]->arrive_and_wait();
    return r;
}

// TMEM scratch (tcgen05.ld/st of the 3D step kernel): 256 doubles per thread, addressed by the 32-bit column index
inline std::vector<double> ark_emu_tmem;
inline double* ark_emu_tm(unsigned a) { return ark_emu_tmem.data() + (size_t)threadIdx.x * 256 + (a & 0xffffu) / 2; }
inline void ark_tm_wait_ld() {}
inline void ark_tm_wait_st() {}
inline void ark_tm_st1(unsigned a, double v0) { ark_emu_tm(a)[0] = v0; }
inline void ark_tm_st4(unsigned a, double v0, double v1, double v2, double v3) { double* p = ark_emu_tm(a); p[0] = v0; p[1] = v1; p[2] = v2; p[3] = v3; }
inline void ark_tm_st8(unsigned a, double v0, double v1, double v2, double v3, double v4, double v5, double v6, double v7) {
    double* p = ark_emu_tm(a); p[0] = v0; p[1] = v1; p[2] = v2; p[3] = v3; p[4] = v4; p[5] = v5; p[6] = v6; p[7] = v7;
}
inline void ark_tm_st2(unsigned a, double v0, double v1) { double* p = ark_emu_tm(a); p[0] = v0; p[1] = v1; }
inline void ark_tm_ld2(unsigned a, double& v0, double& v1) { const double* p = ark_emu_tm(a); v0 = p[0]; v1 = p[1]; }
inline void ark_tm_ld1(unsigned a, double& v0) { v0 = ark_emu_tm(a)[0]; }
inline void ark_tm_ld4(unsigned a, double& v0, double& v1, double& v2, double& v3) { const double* p = ark_emu_tm(a); v0 = p[0]; v1 = p[1]; v2 = p[2]; v3 = p[3]; }
inline void ark_tm_ld8(unsigned a, double& v0, double& v1, double& v2, double& v3, double& v4, double& v5, double& v6, double& v7) {
    const double* p = ark_emu_tm(a); v0 = p[0]; v1 = p[1]; v2 = p[2]; v3 = p[3]; v4 = p[4]; v5 = p[5]; v6 = p[6]; v7 = p[7];
}

inline std::vector<unsigned long long> ark_emu_redu;
inline unsigned long long ark_emu_block_umax(unsigned long long v) {
    ark_emu_redu[threadIdx.x] = v;
    __syncthreads();
    if (threadIdx.x == 0)
        for (unsigned i = 1; i < blockDim.x; ++i) v = std::max(v, ark_emu_redu[i]);
    __syncthreads();
    return v;
}

// run f() for every thread of every block of the grid
inline void ark_emu_launch(emu_dim3 grid, unsigned nthreads, size_t smem_bytes, const std::function<void()>& f,
                           unsigned warp = 32) {
    std::vector<double> smem(smem_bytes / sizeof(double) + 1);
    ark_emu_warp = warp;
    ark_emu_shfl_buf.assign(nthreads, 0.0);
    ark_emu_tmem.assign((size_t)nthreads * 256, 0.0);
    ark_emu_wbar.clear();
    if (nthreads % warp == 0)
        for (unsigned w = 0; w < nthreads / warp; ++w) ark_emu_wbar.emplace_back(std::make_unique<std::barrier<>>(warp));
    ark_emu_smem = smem.data();
    ark_emu_red.assign(nthreads, 0.0);
    ark_emu_redu.assign(nthreads, 0ULL);
    for (unsigned bz = 0; bz < grid.z; ++bz)
        for (unsigned by = 0; by < grid.y; ++by)
            for (unsigned bx = 0; bx < grid.x; ++bx) {
                std::barrier<> bar(nthreads);
                ark_emu_barrier = &bar;
                std::vector<std::thread> th;
                th.reserve(nthreads);
                for (unsigned t = 0; t < nthreads; ++t)
                    th.emplace_back([&, t] {
                        threadIdx.x = t;
                        blockIdx.x = bx; blockIdx.y = by; blockIdx.z = bz;
                        blockDim.x = nthreads;
                        gridDim = grid;
                        f();
                    });
                for (auto& x : th) x.join();
            }
    ark_emu_smem = nullptr;
    ark_emu_barrier = nullptr;
}
