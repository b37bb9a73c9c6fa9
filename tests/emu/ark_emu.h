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
inline void ark_emu_launch(emu_dim3 grid, unsigned nthreads, size_t smem_bytes, const std::function<void()>& f) {
    std::vector<double> smem(smem_bytes / sizeof(double) + 1);
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
