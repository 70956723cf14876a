// ppl_layout.h -- geometry shared by the host planner (ppl_plan.cpp, plain C++: no CUDA call, compiles with g++ alone)
// and the kernels: CTA tile extents, the slab width of PPL_SYM_FULL, and the packed pair indices of the symmetric /
// antisymmetric operands.  Functions are host + device under nvcc, plain inline under g++.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define PPL_HD __host__ __device__ __forceinline__
#else
#define PPL_HD inline
#endif

namespace ppl {

constexpr int BM = 128;      // CTA tile rows
constexpr int BN = 128;      // CTA tile cols
constexpr int BK = 16;       // k per pipeline stage
constexpr int TA_FULL = 16;  // a-block edge of PPL_SYM_FULL: one TMA box row of L, one k-tile of use 2

// Packed column index of the pair (c <= d) / (c < d).  Row c of the triangle is placed so that the index of
// (c,d) has the parity of d (one unused "hole" element every other row; holes are zero in tau+- for good:
// the buffers are cleared once at plan time and no kernel writes a hole).  This makes every run
// (c, d0..d0+15) with d0 even start at an even index, i.e. at a 16-byte aligned address: TMA boxes must
// start 16-byte aligned (an odd FP64 coordinate raises an illegal-instruction error), and PPL_SYM_FULL reads
// such runs of tau+- as k-tiles.  In the minus triangle the element before (c, c+1), c even, is a hole.
PPL_HD int64_t kplus(int c, int d, int v) {
    return (int64_t)c * v - (int64_t)c * (c + 1) / 2 + (c + 1) / 2 + d;
}
PPL_HD int64_t kminus(int c, int d, int v) {
    return (int64_t)c * (2 * v - c - 1) / 2 - c + c / 2 + d;
}
PPL_HD int64_t kplus_extent(int v) { return kplus(v - 1, v - 1, v) + 1; }
PPL_HD int64_t kminus_extent(int v) { return v >= 2 ? kminus(v - 2, v - 1, v) + 1 : 0; }
// packed row index of the occupied pair (i <= j) / (i < j): dense, no holes
PPL_HD int64_t rowplus(int i, int j, int o) { return (int64_t)i * o - (int64_t)i * (i - 1) / 2 + (j - i); }
PPL_HD int64_t rowminus(int i, int j, int o) { return (int64_t)i * (2 * o - i - 1) / 2 + (j - i - 1); }

// Diagonal (b-block == d-block) 16 x 16 blocks of L, packed: only the pairs b_l <= d_l are needed there (the rest is their
// b<->d image), 136 of 256.  k_pack_diag copies them once per apply into Lq[P][blk * 144 + t], t = the row-major index of
// (b_l <= d_l) in the triangle (row b_l holds 16 - b_l entries; t = 136..143 are zero padding): 9 TMA chunks of 16 columns
// per block instead of 16.  Chunk-table entry of a packed chunk: x = -2 - blk, y = its inner coordinate in Lq.
constexpr int DIAG_PACKED = 144, DIAG_PAIRS = 136;
PPL_HD bool diag_unpack(int t, int &bl, int &dl) {
    if (t >= DIAG_PAIRS) return false;
    bl = 0;
    int off = 0;
    while (t - off >= 16 - bl) {
        off += 16 - bl;
        ++bl;
    }
    dl = bl + (t - off);
    return true;
}
}  // namespace ppl
