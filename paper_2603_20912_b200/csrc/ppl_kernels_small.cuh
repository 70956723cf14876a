// ppl_kernels_small.cuh -- the whole ladder in ONE kernel, for launch-bound shapes (nvirt <= 56, nocc <= 8: BASELINE.json's
// tiny and small configs).
//
// At these sizes the tiled path is a chain of 6-34 dependent launches of a few microseconds each, every one far too
// small to fill 148 SMs (tiny: 27 MFLOP; small: W is 63 MB and the step-1 GEMM has 25 rows).  Here one launch does
// step 0, step 1 and the accumulate / mirror of SURVEY 8(a), and the v^4 intermediate never leaves the register file:
//
//   work item = (a; SW consecutive b's), one warp per b.  The CTA stages L[P][a][:] and L[P][b..b+SW)[:] through a
//   cp.async ring, each warp forms  W_ab[c][d] = sum_P L[P,a,c] L[P,b,d]  (eq. 5; 'xac,xbd->acbd') with DMMA
//   m8n8k4 into NB x NB accumulator blocks (NB = ceil(nvirt / 8)), then contracts its W_ab with t2 straight from the
//   accumulators:  R[i,j,a,b] (+)= sum_cd W_ab[c][d] t2[i,j,c,d]  (eq. 4/6; 'acbd,ecfd->efab') -- nocc^2 dot products of
//   FP64 FMAs per lane followed by a fixed-order warp reduction -- and lane 0 writes R[i,j,a,b] and, with pair symmetry,
//   the mirror R[j,i,b,a].  Every R entry is written by exactly one warp: no atomics, bit-reproducible.
//
// Symmetry: with pair-symmetric t2 (every mode but PPL_SYM_NONE) only a <= b is computed (half of nominal, both steps);
// L's own symmetry is not needed and not used.  The S+- packing of the tiled path would save another factor on paper,
// but its fold / two-use bookkeeping is exactly the chain of small launches this kernel exists to avoid.
#pragma once
#include "ppl_device.cuh"

namespace ppl {

constexpr int SMALL_SW = 4;        // warps (= b's) per CTA
constexpr int SMALL_STAGES = 3;
constexpr int SMALL_THREADS = 32 * SMALL_SW;

struct SmallArgs {
    const double *L, *t2;
    double *R;
    int o, v, x;
    int pair;            // 1: items cover a <= b and the mirror entry is written too; 0: every (a, b)
    int nitems;
    double alpha, beta;
    RStrides ts, rs;     // element strides of t2[i,j,c,d] and R[i,j,a,b] (either storage order)
};

template <int NB>
struct SmallCfg {
    static constexpr int W8 = 8 * NB;                      // padded nvirt
    static constexpr int LDA = W8 + 4;                     // [k][c] row stride: 4 mod 8 doubles -> conflict-free LDS.64
    static constexpr int LDB = SMALL_SW * W8 + 4;          // [k][(b_l, d)]
    static constexpr int STAGE = BK * (LDA + LDB);         // doubles
    static constexpr size_t SMEM = (size_t)SMALL_STAGES * STAGE * sizeof(double);
};

// item -> (a, b0): a-major; per a the b's from (pair ? a : 0) in blocks of SW
__device__ __forceinline__ void small_item(int item, int v, int pair, int &a, int &b0) {
    a = 0;
    for (;;) {
        const int nblk = ((pair ? v - a : v) + SMALL_SW - 1) / SMALL_SW;
        if (item < nblk) break;
        item -= nblk;
        ++a;
    }
    b0 = (pair ? a : 0) + item * SMALL_SW;
}

template <int NB>
__global__ void __launch_bounds__(SMALL_THREADS, 2) k_small_fused(const SmallArgs p) {
    using Cfg = SmallCfg<NB>;
    constexpr int W8 = Cfg::W8, LDA = Cfg::LDA, LDB = Cfg::LDB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sm = reinterpret_cast<double *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int v = p.v, vv = v * v;
    const int nkt = (p.x + BK - 1) / BK;
    const int rowlen = v * (1 + SMALL_SW);                 // doubles fetched per P: row a, then rows b0 .. b0+SW-1 (contiguous in L)
    constexpr int MAXR = (W8 * (1 + SMALL_SW) + SMALL_THREADS - 1) / SMALL_THREADS;

    // the padding columns (c, d in [v, 8 NB)) of every stage are never written by a copy: clear them once
    for (int i = tid; i < SMALL_STAGES * Cfg::STAGE; i += SMALL_THREADS) sm[i] = 0.0;
    __syncthreads();

    for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
        int a, b0;
        small_item(item, v, p.pair, a, b0);
        const int nb = min(SMALL_SW, v - b0);              // b's of this item
        // this thread's elements of one P-row of the stage: source offset inside L[P] and destination inside the stage
        int srcoff[MAXR], dstoff[MAXR];
#pragma unroll
        for (int t = 0; t < MAXR; ++t) {
            const int r = tid + t * SMALL_THREADS;
            srcoff[t] = -1;
            dstoff[t] = 0;
            if (r < v) {
                srcoff[t] = a * v + r;
                dstoff[t] = r;
            } else if (r < rowlen) {
                const int s = r - v, bl = s / v, d = s - bl * v;
                if (bl < nb) {
                    srcoff[t] = (b0 + bl) * v + d;
                    dstoff[t] = BK * LDA + bl * W8 + d;
                } else {
                    srcoff[t] = -2;                          // a b beyond nvirt: zeros
                    dstoff[t] = BK * LDA + bl * W8 + d;
                }
            }
        }
        auto load_stage = [&](int kt) {
            double *st = sm + (kt % SMALL_STAGES) * Cfg::STAGE;
            const double *Lp = p.L + (int64_t)kt * BK * vv;
#pragma unroll 1  // (a rolled loop with one running pointer: unrolled, ptxas kept dozens of 64-bit addresses live next to the accumulators)
            for (int k = 0; k < BK; ++k, Lp += vv) {
                const bool inK = kt * BK + k < p.x;
#pragma unroll
                for (int t = 0; t < MAXR; ++t) {
                    if (srcoff[t] == -1) continue;
                    const bool ok = inK && srcoff[t] >= 0;
                    const bool isb = dstoff[t] >= BK * LDA;
                    cp_async8(st + dstoff[t] + k * (isb ? LDB : LDA), ok ? Lp + srcoff[t] : p.L, ok ? 8 : 0);
                }
            }
        };

        double acc[NB][NB][2];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        __syncthreads();  // the previous item's reads of the ring are done
#pragma unroll
        for (int s = 0; s < SMALL_STAGES - 1; ++s) {
            if (s < nkt) load_stage(s);
            cp_async_commit();
        }
        for (int kt = 0; kt < nkt; ++kt) {
            cp_async_wait<SMALL_STAGES - 2>();
            __syncthreads();
            if (kt + SMALL_STAGES - 1 < nkt) load_stage(kt + SMALL_STAGES - 1);
            cp_async_commit();
            const double *as = sm + (kt % SMALL_STAGES) * Cfg::STAGE + g;
            const double *bs = as + BK * LDA + warp * W8;
            if (warp >= nb) continue;  // no b for this warp in a ragged item (it still takes part in the barriers above)
            constexpr int K4_UNROLL = NB >= 6 ? 2 : BK / 4;  // (unrolled, the fragments of all four k-steps are fetched ahead: 4 x 2 NB doubles)
#pragma unroll K4_UNROLL
            for (int k4 = 0; k4 < BK / 4; ++k4) {
                const int kk = k4 * 4 + q;
                double af[NB], bf[NB];
#pragma unroll
                for (int i = 0; i < NB; ++i) af[i] = as[kk * LDA + 8 * i];
#pragma unroll
                for (int j = 0; j < NB; ++j) bf[j] = bs[kk * LDB + 8 * j];
#pragma unroll
                for (int i = 0; i < NB; ++i)
#pragma unroll
                    for (int j = 0; j < NB; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
        }
        cp_async_wait<0>();

        // step 1 from the accumulators: block (i, j): c = 8 i + g, d = 8 j + 2 q, + 1.  Rows / columns >= nvirt of W are exact
        // zeros (zero-padded operands); their t2 addresses are clamped into the array, so they contribute 0 * finite.
        const int b = b0 + warp;
        if (b < v) {
            constexpr int U = NB >= 6 ? 2 : 4;  // (i, j) blocks of t2 per pass (register budget: the accumulators stay live)
            const int oo = p.o * p.o, sa = (int)p.ts.a;
            for (int ij0 = 0; ij0 < oo; ij0 += U) {
                double s[U];
                int64_t tij[U];  // offsets of the (i, j) blocks of t2 (beyond the last one: it is repeated and not stored)
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int ij = min(ij0 + u, oo - 1), i_ = ij / p.o, j_ = ij - i_ * p.o;
                    tij[u] = i_ * p.ts.i + j_ * p.ts.j;
                    s[u] = 0.0;
                }
                // (g, q behind an opaque move: the 2 NB^2 element addresses below are loop-invariant, and hoisted out of this loop
                // they would sit in registers next to the accumulators -- ptxas spilled them; a few integer ops per load are cheaper)
                int g2 = g, q2 = q;
                asm volatile("" : "+r"(g2), "+r"(q2));
#pragma unroll
                for (int i = 0; i < NB; ++i) {
                    const int roff = min(8 * i + g2, v - 1) * sa;
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        const double *e0 = p.t2 + (roff + min(8 * j + 2 * q2, v - 1)), *e1 = p.t2 + (roff + min(8 * j + 2 * q2 + 1, v - 1));
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            s[u] = fma(acc[i][j][0], __ldg(e0 + tij[u]), s[u]);
                            s[u] = fma(acc[i][j][1], __ldg(e1 + tij[u]), s[u]);
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
#pragma unroll
                    for (int m = 16; m >= 1; m >>= 1) s[u] += __shfl_xor_sync(0xffffffffu, s[u], m);
                }
                if (lane == 0) {
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int ij = ij0 + u;
                        if (ij >= oo) break;
                        const int i_ = ij / p.o, j_ = ij - i_ * p.o;
                        r_update(p.R + i_ * p.rs.i + j_ * p.rs.j + a * p.rs.a + b * p.rs.b, s[u], p.alpha, p.beta);
                        if (p.pair && a != b) r_update(p.R + j_ * p.rs.i + i_ * p.rs.j + b * p.rs.a + a * p.rs.b, s[u], p.alpha, p.beta);
                    }
                }
            }
        }
    }
}

}  // namespace ppl
