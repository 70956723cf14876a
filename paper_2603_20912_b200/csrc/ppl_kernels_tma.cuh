// ppl_kernels_tma.cuh -- persistent, warp-specialised sm_100a GEMM kernels for both steps.
//
//   warps 8..11 (warpgroup 2)  : producer warpgroup; gives its registers away (setmaxnreg.dec) and one
//                                elected lane of warp 8 is the TMA producer.  cp.async.bulk.tensor.2d loads 128B-swizzled boxes of
//                                the operands into a TSTAGES-deep shared-memory ring and signals
//                                full[stage] (mbarrier, complete_tx::bytes).
//   warps 0..7                 : consumers.  Wait full[stage], read fragments with conflict-free
//                                LDS.128, issue DMMA m8n8k4 (FP64 tensor pipe), arrive on empty[stage].
//   grid = #SMs, each CTA strides over work items (output tile [, k-split]); the producer runs
//   ahead across item boundaries, so the ring never drains between tiles and the epilogue of one
//   item overlaps the loads of the next.  There is no __syncthreads in the main loop.
//
// Why this shape: ncu on the first (cp.async + __syncthreads) kernels showed the DMMA pipe 86 %
// active; the rest was the per-k-tile address/LDGSTS section executed by all warps in lock step
// behind the barrier and the per-CTA prologue/epilogue at 1 CTA/SM (profiles/r01_*.md).
//
// Shared-memory layouts (TMA SWIZZLE_128B: 16-byte chunk index ^= (128-byte row index & 7)):
//   step 0, operand tile 128 (m) x 16 (k):  8 boxes [mchunk][k=16 rows][16 doubles of m]
//   step 1, operand tile 128 (m) x 16 (k):  1 box   [m=128 rows][16 doubles of k]
// Fragment rows are permuted so that the 8 lanes of a quarter warp hit 8 distinct 16-byte bank
// groups: lane = 4g+q uses row/chunk index c(g) = (g>>1) + 4*(g&1).  The epilogues undo it.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppl_kernels.cuh"

namespace ppl {

constexpr int TSTAGES = 6;
constexpr int CONSUMER_WARPS = 8;
constexpr int TMA_THREADS = 32 * (CONSUMER_WARPS + 4);  // 2 consumer warpgroups + 1 producer warpgroup
constexpr int CONSUMER_REGS = 232, PRODUCER_REGS = 40;  // setmaxnreg: 8*32*232 + 4*32*40 = 64512 <= 65536
constexpr uint32_t TILE_BYTES = BM * BK * sizeof(double);          // one operand tile: 16 KB
constexpr uint32_t STAGE_BYTES = 2 * TILE_BYTES;                   // A + B
constexpr size_t SMEM_TMA = (size_t)TSTAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/;

// ---- mbarrier / TMA primitives (PTX; SASS: SYNCS.*, UTMALDG) ----
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, int c0, int c1, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
// the same with an L2 eviction-priority hint (a createpolicy-encoded 64-bit descriptor: the constants below)
constexpr uint64_t L2_EVICT_NORMAL = 0x1000000000000000ull, L2_EVICT_FIRST = 0x12F0000000000000ull, L2_EVICT_LAST = 0x14F0000000000000ull;
__device__ __forceinline__ void tma_load_2d_hint(void *dst, const CUtensorMap *map, int c0, int c1, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;\n" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(N)); }
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap *map) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(map) : "memory");
}

struct TmaSmem {
    double *a, *b;           // [TSTAGES][BM*BK]
    uint64_t *full, *empty;  // [TSTAGES]
};
__device__ __forceinline__ TmaSmem carve_smem(unsigned char *raw) {
    const uint32_t base = smem_u32(raw);
    unsigned char *al = raw + ((1024u - (base & 1023u)) & 1023u);
    TmaSmem s;
    s.a = reinterpret_cast<double *>(al);
    s.b = reinterpret_cast<double *>(al + (size_t)TSTAGES * TILE_BYTES);
    s.full = reinterpret_cast<uint64_t *>(al + (size_t)TSTAGES * STAGE_BYTES);
    s.empty = s.full + TSTAGES;
    return s;
}
__device__ __forceinline__ void init_barriers(const TmaSmem &s, int tid) {
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < TSTAGES; ++i) {
            mbar_init(&s.full[i], 1);
            mbar_init(&s.empty[i], CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();
}

// Consumer-side release of a ring slot.  The slot read in iteration t is handed back to the producer
// only after the try_wait loop of iteration t+1: warps issue in order, a DMMA cannot issue before the
// LDS that feed it have returned, and every DMMA of iteration t precedes that loop -- so all shared
// loads of the slot are complete when the arrive issues.  (Arriving at the end of iteration t is NOT
// safe: ptxas hoists the arrive above the trailing DMMAs, right behind the last LDS *issue*; with the
// LSU backed up by other warps' epilogue stores the TMA refill then overtook those loads -- caught by
// tests/test_gpu_fullsize.py and reproduced by tests/test_gpu_parity.py::test_persistent_ring_*.)
// The slot of the very last iteration is never released: the producer has nothing left to load.
__device__ __forceinline__ void release_previous(const TmaSmem &sm, int rel_stage, int lane) {
    if (rel_stage >= 0 && lane == 0) mbar_arrive(&sm.empty[rel_stage]);
}

// ---------------------------------------------------------------------------------------------
// step 0 (TMA):  W[(a,b)][(c,d)] = sum_P L[P,a,c] L[P,b,d]      (eq. 5)
// mapL: 2-D tensor {inner = nvirt^2 (a,c flattened), outer = nchol}, box {16, BK}, SWIZZLE_128B.
// ---------------------------------------------------------------------------------------------
struct Step0TmaArgs {
    int a0v, b0v;   // a0*v, b0*v: first flattened (a,c) / (b,d) column of the panels
    int M, N, K;    // ta*v, tb*v, nchol
    int v, tb;
    double *W;
    int64_t ldw;
    double alpha = 1.0, beta = 0.0;  // W = beta W + alpha (product); the ladder path overwrites (1, 0)
};

// mapL / mapB: the row operand and the column operand (the same map twice on the ladder path, where both are L; two
// different tensors when ppl_contract_pair routes a 'k...m...,k...n...->m...n...' contraction here: with v = N, tb = 1,
// ldw = N^2 the store address a_l tb ldw + c v + b_l ldw + d is m N + n, a dense row-major C[M][N])
__global__ void __launch_bounds__(TMA_THREADS, 1)
    k_step0_tma(const __grid_constant__ CUtensorMap mapL, const __grid_constant__ CUtensorMap mapB, const Step0TmaArgs p) {
    extern __shared__ unsigned char smem_raw[];
    const TmaSmem sm = carve_smem(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    init_barriers(sm, tid);

    const int tiles_m = (p.M + BM - 1) / BM, tiles_n = (p.N + BN - 1) / BN;
    const int num_items = tiles_m * tiles_n;
    const int nkt = (p.K + BK - 1) / BK;

    if (warp >= CONSUMER_WARPS) {
        // ================================ producer warpgroup ================================
        setmaxnreg_dec<PRODUCER_REGS>();
        if (warp == CONSUMER_WARPS && lane == 0) {
            prefetch_tmap(&mapL);
            prefetch_tmap(&mapB);
            int stage = 0;
            uint32_t phase = 0;
            for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
                int tm, tn;
                raster(item, tiles_m, tiles_n, tm, tn);
                const int xa = p.a0v + tm * BM, xb = p.b0v + tn * BN;
                for (int kt = 0; kt < nkt; ++kt) {
                    mbar_wait(&sm.empty[stage], phase ^ 1);
                    mbar_expect_tx(&sm.full[stage], STAGE_BYTES);
                    double *da = sm.a + (size_t)stage * BM * BK, *db = sm.b + (size_t)stage * BN * BK;
#pragma unroll
                    for (int i = 0; i < BM / 16; ++i) tma_load_2d(da + i * BK * 16, &mapL, xa + 16 * i, kt * BK, &sm.full[stage]);
#pragma unroll
                    for (int i = 0; i < BN / 16; ++i) tma_load_2d(db + i * BK * 16, &mapB, xb + 16 * i, kt * BK, &sm.full[stage]);
                    if (++stage == TSTAGES) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
        return;
    }
    // ================================ consumers ================================
    setmaxnreg_inc<CONSUMER_REGS>();
    const int g = lane >> 2, q = lane & 3;
    const int c = (g >> 1) + 4 * (g & 1);  // permuted row/chunk index of this lane's fragment row
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    // fragment offsets (doubles) inside an operand tile for k4 even / odd: row k = 4*k4 + q
    const int offk_even = q * 16 + ((c ^ q) << 1);
    const int offk_odd = (q + 4) * 16 + ((c ^ (q + 4)) << 1);
    int stage = 0, rel_stage = -1;
    uint32_t phase = 0;
    for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
        int tm, tn;
        raster(item, tiles_m, tiles_n, tm, tn);
        const int m0 = tm * BM, n0 = tn * BN;
        double acc[8][4][2];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        for (int kt = 0; kt < nkt; ++kt) {
            mbar_wait(&sm.full[stage], phase);
            release_previous(sm, rel_stage, lane);
            const double *as = sm.a + (size_t)stage * BM * BK + (wm * 4) * (BK * 16);
            const double *bs = sm.b + (size_t)stage * BN * BK + (wn * 2) * (BK * 16);
#pragma unroll
            for (int k4 = 0; k4 < BK / 4; ++k4) {
                const int off = (k4 >> 1) * 128 + ((k4 & 1) ? offk_odd : offk_even);
                double2 a[4], b[2];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = *reinterpret_cast<const double2 *>(as + i * (BK * 16) + off);
#pragma unroll
                for (int j = 0; j < 2; ++j) b[j] = *reinterpret_cast<const double2 *>(bs + j * (BK * 16) + off);
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        dmma(acc[2 * i][2 * j][0], acc[2 * i][2 * j][1], a[i].x, b[j].x);
                        dmma(acc[2 * i][2 * j + 1][0], acc[2 * i][2 * j + 1][1], a[i].x, b[j].y);
                        dmma(acc[2 * i + 1][2 * j][0], acc[2 * i + 1][2 * j][1], a[i].y, b[j].x);
                        dmma(acc[2 * i + 1][2 * j + 1][0], acc[2 * i + 1][2 * j + 1][1], a[i].y, b[j].y);
                    }
            }
            rel_stage = stage;  // released after the NEXT stage's wait (see release_previous)
            if (++stage == TSTAGES) {
                stage = 0;
                phase ^= 1;
            }
        }
        // epilogue.  block (2i+e, 2j+f): frag row g <-> m = mw + 16i + 2c(g) + e;
        //   c0 <-> n = nw + 16j + 2q + f,   c1 <-> n = nw + 16j + 2q + 8 + f
        const int v = p.v;
        const bool pair_ok = (v & 1) == 0;  // n even & v even: (n, n+1) share one b and are 16-byte aligned
        const bool plain = p.alpha == 1.0 && p.beta == 0.0;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int m = m0 + wm * WTM + 16 * i + 2 * c + e;
                if (m >= p.M) continue;
                const int al = m / v, cc = m - al * v;
                double *wrow = p.W + (int64_t)al * p.tb * p.ldw + (int64_t)cc * v;
#pragma unroll
                for (int j = 0; j < 2; ++j)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {  // h = 0: c0 values, h = 1: c1 values
                        const int n = n0 + wn * WTN + 16 * j + 2 * q + 8 * h;
                        const double v0 = acc[2 * i + e][2 * j][h], v1 = acc[2 * i + e][2 * j + 1][h];
                        const int bl = n / v, d = n - bl * v;
                        if (plain && pair_ok && n + 1 < p.N) {
                            *reinterpret_cast<double2 *>(wrow + (int64_t)bl * p.ldw + d) = make_double2(v0, v1);
                        } else {
                            if (n < p.N) r_update(wrow + (int64_t)bl * p.ldw + d, v0, p.alpha, p.beta);
                            if (n + 1 < p.N) {
                                const int bl1 = (n + 1) / v, d1 = (n + 1) - bl1 * v;
                                r_update(wrow + (int64_t)bl1 * p.ldw + d1, v1, p.alpha, p.beta);
                            }
                        }
                    }
            }
    }
}

// ---------------------------------------------------------------------------------------------
// step 1 (TMA):  part[z][(i,j)][(a,b)] = sum_{(c,d) in split z} t2[(i,j)][(c,d)] W[(a,b)][(c,d)]
// mapA: t2 as {inner = nvirt^2, outer = nocc^2}, box {16, 16*NI};  mapB: W slot as {inner = nvirt^2,
// outer = T*T}, box {16, 128}; SWIZZLE_128B.
// NI = maximum number of 8-row blocks per warp along M (TMA box of A: 16*NI rows); see MSplit below.
// ---------------------------------------------------------------------------------------------
// Rows of the M side (nocc^2, or the packed (i<=j) / (i<j) rows) are cut into 8-row blocks and dealt to 2*tiles_m
// "half-tiles" -- the two warp rows of a CTA tile -- of `base` or `base + 1` blocks (the first `rem` get the extra one).
// nocc^2-like extents are rarely a multiple of a CTA tile height (820, 780, 1830, 210 ...): with uniform tiles of
// 16*NI rows the padding was 3-5 % of the DMMA work of step 1; this way it is < 8 rows in all.  Each SMSP hosts one
// warp of either warp row, so a CTA tile costs ni0 + ni1 blocks on every SMSP: tiles differ by at most 2 in 2*NI.
struct MSplit {
    int tiles_m, base, rem;
};
__device__ __forceinline__ void m_tile(const MSplit &g, int tm, int &row0, int &ni0, int &ni1) {
    const int h = 2 * tm;
    ni0 = g.base + (h < g.rem ? 1 : 0);
    ni1 = g.base + (h + 1 < g.rem ? 1 : 0);
    row0 = 8 * (h * g.base + min(h, g.rem));
}

struct Step1TmaArgs {
    int M, N, K;      // nocc^2, ta*tb, nvirt^2 (K = END of the contraction range)
    int k0;           // first k of the contraction range (0 except in PPL_SYM_FULL; any value: TMA boxes may start anywhere)
    int k_per_split;  // multiple of BK
    int splitk;
    MSplit ms;
    double *part;     // [splitk][M][N]
};

template <int NI>
struct Step1Cfg {
    static constexpr int BM1 = 16 * NI;                                   // CTA tile rows (TMA box; a tile uses 8*(ni0+ni1) of them)
    static constexpr uint32_t A_BYTES = BM1 * BK * sizeof(double);
    static constexpr uint32_t STAGE = A_BYTES + TILE_BYTES;               // A + B(128 x 16)
    static constexpr size_t SMEM = (size_t)TSTAGES * STAGE + 1024 + 256;
};

// The k loop of one work item of step 1 for a warp that owns NA (= NI or NI - 1) 8-row blocks.
// as_off / bs_off: the warp's first row inside the A / B stage tile.
template <int NI, int NA>
__device__ __forceinline__ void step1_consume(double (&acc)[NI][4][2], const TmaSmem &sm, int as_off, int bs_off, int off0, int off1,
                                              int nkt, int nact, int &stage, uint32_t &phase, int &rel_stage, int lane) {
    constexpr int BM1 = Step1Cfg<NI>::BM1;
    for (int kt = 0; kt < nkt; ++kt) {
        mbar_wait(&sm.full[stage], phase);
        release_previous(sm, rel_stage, lane);
        const double *as = sm.a + (size_t)stage * BM1 * BK + as_off;
        const double *bs = sm.b + (size_t)stage * BN * BK + bs_off;
#pragma unroll
        for (int k8 = 0; k8 < BK / 8; ++k8) {
            const int off = k8 ? off1 : off0;
            double2 a[NA > 0 ? NA : 1], b[4];
#pragma unroll
            for (int i = 0; i < NA; ++i)
                a[i] = *reinterpret_cast<const double2 *>(as + i * 8 * BK + off);
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = *reinterpret_cast<const double2 *>(bs + j * 8 * BK + off);
#pragma unroll
            for (int i = 0; i < NA; ++i)
                {
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
                }
#pragma unroll
            for (int i = 0; i < NA; ++i)
                {
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
                }
        }
        rel_stage = stage;  // released after the NEXT stage's wait (see release_previous)
        if (++stage == TSTAGES) {
            stage = 0;
            phase ^= 1;
        }
    }
}

template <int NI>
__global__ void __launch_bounds__(TMA_THREADS, 1)
    k_step1_tma(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const Step1TmaArgs p) {
    using Cfg = Step1Cfg<NI>;
    constexpr int BM1 = Cfg::BM1;
    extern __shared__ unsigned char smem_raw[];
    // ring: [TSTAGES] A tiles, then [TSTAGES] B tiles, then the barriers
    const uint32_t base = smem_u32(smem_raw);
    unsigned char *al = smem_raw + ((1024u - (base & 1023u)) & 1023u);
    TmaSmem sm;
    sm.a = reinterpret_cast<double *>(al);
    sm.b = reinterpret_cast<double *>(al + (size_t)TSTAGES * Cfg::A_BYTES);
    sm.full = reinterpret_cast<uint64_t *>(al + (size_t)TSTAGES * Cfg::STAGE);
    sm.empty = sm.full + TSTAGES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    init_barriers(sm, tid);

    const int tiles_m = p.ms.tiles_m, tiles_n = (p.N + BN - 1) / BN;
    const int tiles_mn = tiles_m * tiles_n;
    const int num_items = tiles_mn * p.splitk;

    if (warp >= CONSUMER_WARPS) {
        setmaxnreg_dec<PRODUCER_REGS>();
        if (warp == CONSUMER_WARPS && lane == 0) {
            prefetch_tmap(&mapA);
            prefetch_tmap(&mapB);
            int stage = 0;
            uint32_t phase = 0;
            for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
                const int z = item / tiles_mn, r = item - z * tiles_mn;
                const int tm = r % tiles_m, tn = r / tiles_m;
                int row0, ni0, ni1;
                m_tile(p.ms, tm, row0, ni0, ni1);
                const int kbeg = p.k0 + z * p.k_per_split, kend = min(p.K, kbeg + p.k_per_split);
                for (int k = kbeg; k < kend; k += BK) {
                    mbar_wait(&sm.empty[stage], phase ^ 1);
                    mbar_expect_tx(&sm.full[stage], Cfg::STAGE);
                    tma_load_2d(sm.a + (size_t)stage * BM1 * BK, &mapA, k, row0, &sm.full[stage]);
                    tma_load_2d(sm.b + (size_t)stage * BN * BK, &mapB, k, tn * BN, &sm.full[stage]);
                    if (++stage == TSTAGES) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
        return;
    }
    setmaxnreg_inc<CONSUMER_REGS>();
    const int g = lane >> 2, q = lane & 3;
    const int c = (g >> 1) + 4 * (g & 1);
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    // row r = 8i + c, 16-byte chunk (k8*4 + q) ^ c
    const int off0 = c * 16 + ((q ^ c) << 1);
    const int off1 = c * 16 + (((4 + q) ^ c) << 1);
    int stage = 0, rel_stage = -1;
    uint32_t phase = 0;
    for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
        const int z = item / tiles_mn, r = item - z * tiles_mn;
        const int tm = r % tiles_m;
        int row0, ni0, ni1;
        m_tile(p.ms, tm, row0, ni0, ni1);
        const int nact = wm ? ni1 : ni0;          // 8-row blocks of this warp
        const int wrow = wm ? 8 * ni0 : 0;        // its first row inside the CTA tile
        const int kbeg = p.k0 + z * p.k_per_split, kend = min(p.K, kbeg + p.k_per_split);
        const int nkt = max(0, (kend - kbeg + BK - 1) / BK);
        double acc[NI][4][2];
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        if (nact == NI)
            step1_consume<NI, NI>(acc, sm, wrow * BK, (wn * WTN) * BK, off0, off1, nkt, nact, stage, phase, rel_stage, lane);
        else  // nact == NI - 1: the host's row tiling hands a warp NI or NI - 1 blocks, nothing else (m_geom_tma)
            step1_consume<NI, NI - 1>(acc, sm, wrow * BK, (wn * WTN) * BK, off0, off1, nkt, nact, stage, phase, rel_stage, lane);

        // epilogue: block (i,j): frag row g <-> m = row0 + wrow + 8i + c(g); c0 <-> n = nw + 8j + q, c1 <-> n + 4
        // (the tile coordinates are derived again from the item number behind an opaque move, so that none of them
        // stays live across the k loop: the NI = 10 instance has no register to spare)
        int it2 = item;
        asm volatile("" : "+r"(it2));
        const int z2 = it2 / tiles_mn, r2 = it2 - z2 * tiles_mn;
        int erow0, eni0, eni1;
        m_tile(p.ms, r2 % tiles_m, erow0, eni0, eni1);
        const int enact = wm ? eni1 : eni0, en0 = (r2 / tiles_m) * BN;
        erow0 += wm ? 8 * eni0 : 0;
        double *part = p.part + (int64_t)z2 * p.M * p.N;
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const int m = erow0 + 8 * i + c;
            if (i >= enact || m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int n = en0 + wn * WTN + 8 * j + q;
                double *dst = part + (int64_t)m * p.N + n;
                if (n < p.N) dst[0] = acc[i][j][0];
                if (n + 4 < p.N) dst[4] = acc[i][j][1];
            }
        }
    }
}

}  // namespace ppl
