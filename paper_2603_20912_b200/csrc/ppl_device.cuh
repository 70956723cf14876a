// ppl_device.cuh -- device-side primitives shared by the translation units of libppl: tile constants, the FP64 tensor
// MMA (DMMA m8n8k4), cp.async copies, the grouped tile raster and the R update.  Only constexpr values and
// __device__ __forceinline__ functions: safe to include from several .cu files (the __global__ kernels are not here).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppl_layout.h"

namespace ppl {

constexpr int STAGES = 4;    // cp.async ring depth
constexpr int NTHREADS = 256;
constexpr int WARPS_N = 4;   // 2 (m) x 4 (n) warps, warp tile 64 x 32
constexpr int WTM = 64, WTN = 32;
constexpr int PADMN = 4;     // row padding (doubles) of the MN-contiguous smem layout
constexpr int LDS_MN = BM + PADMN;
constexpr int GROUP_M = 12;  // raster group: a wave of 148 CTAs covers ~12 x 12 tiles (L2 reuse)

constexpr size_t SMEM_MN = (size_t)STAGES * BK * (LDS_MN + LDS_MN) * sizeof(double);
constexpr size_t SMEM_K = (size_t)STAGES * (BM + BN) * BK * sizeof(double);

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// zero-filling async copies: bytes beyond src_bytes are written as 0 (tile edges, k tail)
__device__ __forceinline__ void cp_async16(void *dst, const void *src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_u32(dst)), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void *dst, const void *src, int src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(smem_u32(dst)), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// tile index -> (tm, tn) with grouped rasterisation
__device__ __forceinline__ void raster(int pid, int tiles_m, int tiles_n, int &tm, int &tn, int group_m = GROUP_M) {
    const int per_group = group_m * tiles_n;
    const int gid = pid / per_group;
    const int first_m = gid * group_m;
    const int gsize = min(tiles_m - first_m, group_m);
    const int r = pid - gid * per_group;
    tm = first_m + r % gsize;
    tn = r / gsize;
}

struct RStrides {
    int64_t i, j, a, b;  // element strides of R[i,j,a,b]
};

__device__ __forceinline__ void r_update(double *r, double val, double alpha, double beta) {
    *r = (beta == 0.0) ? alpha * val : beta * (*r) + alpha * val;
}

}  // namespace ppl
