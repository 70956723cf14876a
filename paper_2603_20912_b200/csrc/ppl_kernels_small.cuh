// ppl_kernels_small.cuh -- the whole ladder in ONE kernel, for launch-bound shapes (nvirt <= 56, nocc <= 8: BASELINE.json's
// tiny and small configs).
//
// At these sizes the tiled path is a chain of 6-34 dependent launches of a few microseconds each, every one far too
// small to fill 148 SMs (tiny: 27 MFLOP; small: W is 63 MB and the step-1 GEMM has 25 rows).  Here one launch does
// step 0, step 1 and the accumulate / mirror of SURVEY 8(a), and the v^4 intermediate never leaves the register file:
//
//   work item = (a; SW consecutive b's), one warp per b.  Rows L[P][a][:] and L[P][b .. b+SW)[:] of 16 P's at a time are
//   brought into a 3-stage shared-memory ring by TMA bulk copies (cp.async.bulk, one per row block, mbarrier complete_tx;
//   SASS UBLKCP) issued by lane 0 of each warp; each warp forms  W_ab[c][d] = sum_P L[P,a,c] L[P,b,d]  (eq. 5,
//   PAPER.md:63; 'xac,xbd->acbd') with DMMA m8n8k4 into NB x NB accumulator blocks (NB = ceil(nvirt / 8)), then contracts
//   its W_ab with t2 straight from the accumulators:  R[i,j,a,b] (+)= sum_cd W_ab[c][d] t2[i,j,c,d]  (eq. 4/6;
//   'acbd,ecfd->efab') -- nocc^2 dot products of FP64 FMAs per lane against t2 blocks staged through the same shared
//   memory (one bulk copy per (i,j) block, two blocks at a time, double-buffered, shared by the CTA's warps), followed by
//   a fixed-order warp reduction -- and lane 0 writes R[i,j,a,b] and, with pair symmetry, the mirror R[j,i,b,a].  Every
//   R entry is written by exactly one warp: no atomics, bit-reproducible.
//
// Bulk copies need 16-byte aligned rows: for odd nvirt (or a t2 stored 'iajb', or misaligned buffers) k_small_prepack
// first copies L and t2 into plan-owned buffers with rows padded to an even length (one extra launch of a few
// microseconds).  Earlier forms of this kernel, measured at the small config: element-wise 8-byte cp.async gathers with t2
// read from global memory in step 1 -- 661 us, 12 of 13 stall samples on the long scoreboard; t2 staged through shared
// memory -- 342 us, 82 M warp instructions for 4 M DMMAs, i.e. issue-bound on address arithmetic at 1-2 warps per scheduler
// (the tiled path: 261 us).
//
// Symmetry: with pair-symmetric t2 (every mode but PPL_SYM_NONE) only a <= b is computed (half of nominal, both steps);
// L's own symmetry is not needed and not used.  The S+- packing of the tiled path would save another factor on paper,
// but its fold / two-use bookkeeping is exactly the chain of small launches this kernel exists to avoid.
#pragma once
#include "ppl_kernels.cuh"

namespace ppl {

constexpr int SMALL_SW = 4;        // warps (= b's) per CTA
constexpr int SMALL_STAGES = 3;
constexpr int SMALL_THREADS = 32 * SMALL_SW;
constexpr int SMALL_MAX_OO = 64;   // nocc <= 8
constexpr int SMALL_MAX_STAGES = 8;

struct SmallArgs {
    const double *L;     // [x][v][ldl] (ldl even, 16-byte aligned: the caller's L, or the padded copy)
    const double *t2;    // [o*o][v][ldt] in (i,j) order (ldt even, aligned: the caller's t2, or the padded / re-ordered copy)
    double *R;
    int o, v, x;
    int ldl, ldt;
    int pair;            // 1: items cover a <= b and the mirror entry is written too; 0: every (a, b)
    int nitems;
    double alpha, beta;
    RStrides rs;         // element strides of R[i,j,a,b] (either storage order)
    // PPL_OPT_VERIFY_INPUTS = 1 without a launch of its own: the first `ncheck` CTAs scan the inputs for the symmetry the plan's
    // mode relies on (check_inputs_scan) instead of taking work items; flags and, from the last of them to finish, the
    // sequence number `seq` go to mapped pinned host memory (chk.flags[0..1], chk.flags[4]), where the next call on the plan
    // reads them.  The work items run on the other CTAs meanwhile.
    CheckArgs chk;
    int ncheck;
    int seq;
    int *done;           // device counter of finished check CTAs (zero between launches)
    // 1: all of t2 (nocc^2 blocks of nvirt x ldt doubles) is staged ONCE per CTA into a region of its own behind the ring, by
    // bulk copies issued before the k loop: step 1 then waits for nothing and makes one pass.  The host sets it when every
    // CTA has a single work item and the region fits (the tiny config: 80 KB) -- there the 4-5 dependent copy latencies of
    // the passes were a third of the kernel.
    int t2_resident;
    int nstages;         // k-loop ring depth: SMALL_STAGES, or nchol / 16 + 1 (<= SMALL_MAX_STAGES) where a CTA has one item and the
                         // shared memory to spare: every row of L the item needs is then in flight at once (tiny: one copy latency, not two)
};

template <int NB>
struct SmallCfg {
    static constexpr int W8 = 8 * NB;                      // padded nvirt
    static constexpr int LDA = W8 + 4;                     // [k][c] row stride: 4 mod 8 doubles -> conflict-free LDS.64
    static constexpr int LDB = SMALL_SW * W8 + 4;          // [k][(b_l, d)]: the SW rows of one P are contiguous, ldl apart
    static constexpr int STAGE = BK * (LDA + LDB);         // doubles
    static constexpr int RING = SMALL_STAGES * STAGE;      // the default ring (the host may ask for up to SMALL_MAX_STAGES stages)
    static constexpr int LDT = W8 + ((NB & 1) ? 0 : 8);    // row stride of the padded copy of t2: 8 (mod 16) doubles (see step 1)
    // ring, then 16 doubles for the mbarriers (<= SMALL_MAX_STAGES + 3), then the warps' results
    __host__ __device__ static constexpr size_t smem(int nstages) {
        return ((size_t)nstages * STAGE + 16 + (size_t)SMALL_SW * SMALL_MAX_OO) * sizeof(double);
    }
    static constexpr size_t SMEM = smem(SMALL_STAGES);
};

// ---- mbarrier / bulk-copy primitives (as in ppl_kernels_tma.cuh; repeated here so that this header stands alone) ----
__device__ __forceinline__ void sm_mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void sm_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sm_mbar_wait(uint64_t *bar, uint32_t parity) {
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
__device__ __forceinline__ void sm_bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

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
    constexpr int LDA = Cfg::LDA, LDB = Cfg::LDB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sm = reinterpret_cast<double *>(smem_raw);
    const int nst = p.nstages, RING = nst * Cfg::STAGE;
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + RING);  // [nst] k-loop stages, then [2] t2 halves, then [1]: all of t2 (t2_resident)
    uint64_t *tfull = full + nst;
    double *results = sm + RING + 16;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if ((int)blockIdx.x < p.ncheck) {  // a check CTA (see SmallArgs)
        const int f = check_inputs_scan(p.chk, reinterpret_cast<double(*)[33]>(sm), blockIdx.x, p.ncheck);
        if (f & 1) p.chk.flags[0] = 1;
        if (f & 2) p.chk.flags[1] = 1;
        __threadfence_system();  // the flags are on their way before this CTA counts as done
        __syncthreads();
        if (tid == 0 && atomicAdd(p.done, 1) == p.ncheck - 1) {
            *p.done = 0;
            __threadfence_system();
            p.chk.flags[4] = p.seq;
        }
        return;
    }
    const int g = lane >> 2, q = lane & 3;
    const int v = p.v, ldl = p.ldl, ldt = p.ldt;
    const int64_t lstride = (int64_t)v * ldl;              // doubles between L[P] and L[P+1]
    const int nkt = (p.x + BK - 1) / BK;

    // Everything a fragment may touch beyond what a copy wrote (columns >= ldl of a row, rows of an absent b, the k tail)
    // must hold FINITE values: it meets exact zeros or is masked out below.  Clear the ring once.
    for (int i = tid; i < RING; i += SMALL_THREADS) sm[i] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) sm_mbar_init(&full[s], SMALL_SW);
        sm_mbar_init(&tfull[0], 1);
        sm_mbar_init(&tfull[1], 1);
        sm_mbar_init(&tfull[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // the generic-proxy clears above precede the bulk copies below
    __syncthreads();
    uint32_t phbits = 0, tphbits = 0;  // phase parity of every barrier, one bit each
    double *tres = results + SMALL_SW * SMALL_MAX_OO;  // t2_resident: nocc^2 blocks, then a cleared pad (reads past the last block)
    bool t2_here = false;
    if (p.t2_resident) {
        const int oo_ = p.o * p.o, tblk_ = v * ldt;
        for (int i = tid; i < 8 * NB * ldt + 8 * NB; i += SMALL_THREADS) tres[oo_ * tblk_ + i] = 0.0;
        if (tid == 0) {
            sm_mbar_expect_tx(&tfull[2], (uint32_t)oo_ * tblk_ * 8);
            for (int u = 0; u < oo_; ++u) sm_bulk_g2s(tres + u * tblk_, p.t2 + (int64_t)u * tblk_, (uint32_t)tblk_ * 8, &tfull[2]);
        }
    }

    for (int item = blockIdx.x - p.ncheck; item < p.nitems; item += gridDim.x - p.ncheck) {
        int a, b0;
        small_item(item, v, p.pair, a, b0);
        const int nb = min(SMALL_SW, v - b0);              // b's of this item
        // stage kt: rows P = 16 kt .. 16 kt + 15 (those below nchol); warp w issues the copies of k = w, w + SW, ...
        auto load_stage = [&](int kt) {
            if (lane != 0) return;
            const int s = kt % nst;
            double *st = sm + s * Cfg::STAGE;
            const uint32_t abytes = (uint32_t)ldl * 8, bbytes = (uint32_t)nb * ldl * 8;
            int rows = 0;
            for (int k = warp; k < BK; k += SMALL_SW) rows += (kt * BK + k < p.x) ? 1 : 0;
            sm_mbar_expect_tx(&full[s], rows * (abytes + bbytes));
            for (int k = warp; k < BK; k += SMALL_SW) {
                const int P = kt * BK + k;
                if (P >= p.x) break;
                const double *Lp = p.L + P * lstride;
                sm_bulk_g2s(st + k * LDA, Lp + (int64_t)a * ldl, abytes, &full[s]);
                sm_bulk_g2s(st + BK * LDA + k * LDB, Lp + (int64_t)b0 * ldl, bbytes, &full[s]);
            }
        };

        // small accumulator files have registers to spare: the old R values this warp will update are fetched now, so that their
        // (cold) global-memory latency runs under the k loop instead of behind step 1
        constexpr int PREFETCH_R_MAX_NB = 4;
        double rold[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
        if (NB <= PREFETCH_R_MAX_NB && p.beta != 0.0 && b0 + warp < v) {
            const int b_ = b0 + warp;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int ij = lane + 32 * t;
                if (ij >= p.o * p.o) break;
                const int i_ = ij / p.o, j_ = ij - i_ * p.o;
                rold[t][0] = p.R[i_ * p.rs.i + j_ * p.rs.j + a * p.rs.a + b_ * p.rs.b];
                if (p.pair && a != b_) rold[t][1] = p.R[j_ * p.rs.i + i_ * p.rs.j + b_ * p.rs.a + a * p.rs.b];
            }
        }

        double acc[NB][NB][2];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        __syncthreads();  // the previous item's reads of the ring are done
        for (int s = 0; s < nst - 1; ++s)
            if (s < nkt) load_stage(s);
        for (int kt = 0; kt < nkt; ++kt) {
            const int s = kt % nst;
            sm_mbar_wait(&full[s], (phbits >> s) & 1u);
            phbits ^= 1u << s;
            __syncthreads();  // every warp has finished stage kt - 1: its slot may be refilled
            if (kt + nst - 1 < nkt) load_stage(kt + nst - 1);
            if (warp >= nb) continue;  // no b for this warp in a ragged item (it still takes part in the barriers)
            const int kvalid = min(BK, p.x - kt * BK);     // the k tail of the last stage holds rows of an older stage: skip them
            const double *as = sm + s * Cfg::STAGE + g;
            const double *bs = sm + s * Cfg::STAGE + BK * LDA + warp * ldl + g;
            constexpr int K4_UNROLL = NB >= 6 ? 2 : BK / 4;  // (unrolled further, the fragments of all four k-steps are fetched ahead)
#pragma unroll K4_UNROLL
            for (int k4 = 0; k4 < BK / 4; ++k4) {
                if (k4 * 4 >= kvalid) break;
                const int kk = k4 * 4 + q;
                const bool live = kk < kvalid;
                double af[NB], bf[NB];
#pragma unroll
                for (int i = 0; i < NB; ++i) af[i] = live ? as[kk * LDA + 8 * i] : 0.0;
#pragma unroll
                for (int j = 0; j < NB; ++j) bf[j] = bs[kk * LDB + 8 * j];
#pragma unroll
                for (int i = 0; i < NB; ++i)
#pragma unroll
                    for (int j = 0; j < NB; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
        }
        // rows c >= nvirt and columns d >= nvirt of the blocks were fed from beyond the rows (finite, but not W): drop them
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                const bool rok = 8 * i + g < v;
                if (!rok || 8 * j + 2 * q >= v) acc[i][j][0] = 0.0;
                if (!rok || 8 * j + 2 * q + 1 >= v) acc[i][j][1] = 0.0;
            }

        // ---- step 1 from the accumulators.  W_ab block (i, j) holds c = 8 i + g, d = 8 j + 2 q, + 1.  The (i', j') blocks of t2
        // ([nvirt][ldt] doubles each, contiguous) come in by one bulk copy each, several per pass, double-buffered, and are
        // read back as 16-byte pairs (d, d + 1).  With ldt = 8 (mod 16) -- what the padded copy of k_small_prepack has, and an
        // un-padded t2 with nvirt = 8 (mod 16) -- the pairs a quarter warp reads (two consecutive g's, q = 0..3) fall into eight
        // different bank groups; at other strides some of them collide (ncu, nvirt = 53 at stride 54: half of the step's
        // shared-memory wavefronts).  Whatever a pair reads beyond a block's rows / columns is finite and meets a zero of W.
        __syncthreads();  // every warp has left the k loop: the ring is free
        const int b = b0 + warp;
        const int oo = p.o * p.o;
        const int LDT = ldt;
        const int tblk = v * ldt;                             // doubles per staged block
        // blocks per pass: as many as two halves of the ring hold (a fragment pair may read up to 8 NB rows / columns into what
        // follows its block, which must stay inside the ring)
        const bool resident = p.t2_resident != 0;
        const int bpp = resident ? oo : max(1, min(8, ((RING - (8 * NB - 1) * ldt - 8 * NB) / tblk + 1) / 2));
        const int npass = (oo + bpp - 1) / bpp;
        if (resident && !t2_here) {
            sm_mbar_wait(&tfull[2], 0);
            t2_here = true;
        }
        auto load_pass = [&](int ps) {                        // blocks bpp ps ... into half (ps & 1)
            if (tid != 0) return;
            const int h = ps & 1, n = min(bpp, oo - bpp * ps);
            sm_mbar_expect_tx(&tfull[h], (uint32_t)n * tblk * 8);
            for (int u = 0; u < n; ++u)
                sm_bulk_g2s(sm + (h * bpp + u) * tblk, p.t2 + (int64_t)(bpp * ps + u) * tblk, (uint32_t)tblk * 8, &tfull[h]);
        };
        if (!resident) load_pass(0);
        double *res = results + warp * SMALL_MAX_OO;  // this warp's nocc^2 results
        for (int ps = 0; ps < npass; ++ps) {
            const int h = ps & 1;
            if (!resident) {
                if (ps + 1 < npass) load_pass(ps + 1);        // (its half was read in pass ps - 1: the barrier below, last iteration)
                sm_mbar_wait(&tfull[h], (tphbits >> h) & 1u);
                tphbits ^= 1u << h;
            }
            const double *tbase = resident ? tres : sm + h * bpp * tblk;
            if (b < v) {
                const int n = min(bpp, oo - bpp * ps);
                for (int u0 = 0; u0 < n; u0 += 2) {           // two blocks at a time: four independent FMA chains
                    double s[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
                    const int u1 = min(u0 + 1, n - 1);        // (an odd last block is read twice and stored once)
                    const double *t0 = tbase + u0 * tblk + g * LDT + 2 * q;
                    const int du = (u1 - u0) * tblk;
#pragma unroll
                    for (int i = 0; i < NB; ++i)
#pragma unroll
                        for (int j = 0; j < NB; ++j) {
                            const double2 ta = *reinterpret_cast<const double2 *>(t0 + 8 * i * LDT + 8 * j);
                            const double2 tb = *reinterpret_cast<const double2 *>(t0 + du + 8 * i * LDT + 8 * j);
                            s[0][0] = fma(acc[i][j][0], ta.x, s[0][0]);
                            s[0][1] = fma(acc[i][j][1], ta.y, s[0][1]);
                            s[1][0] = fma(acc[i][j][0], tb.x, s[1][0]);
                            s[1][1] = fma(acc[i][j][1], tb.y, s[1][1]);
                        }
                    double r[2] = {s[0][0] + s[0][1], s[1][0] + s[1][1]};
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
#pragma unroll
                        for (int m = 16; m >= 1; m >>= 1) r[u] += __shfl_xor_sync(0xffffffffu, r[u], m);
                    }
                    if (lane < 2 && u0 + lane < n) res[bpp * ps + u0 + lane] = lane ? r[1] : r[0];
                }
            }
            if (!resident) __syncthreads();  // pass ps has been read: its half may be refilled
        }
        // R[i,j,a,b] (and the mirror): one (i,j) per lane, so that the read-modify-writes of a warp are in flight together
        // (one result at a time from lane 0, each behind its own global load, was 40 % of the stall samples at tiny)
        if (b < v) {
            __syncwarp();
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int ij = lane + 32 * t;
                if (ij >= oo) break;
                const int i_ = ij / p.o, j_ = ij - i_ * p.o;
                const double val = res[ij];
                double *rd = p.R + i_ * p.rs.i + j_ * p.rs.j + a * p.rs.a + b * p.rs.b;
                double *rm = p.R + j_ * p.rs.i + i_ * p.rs.j + b * p.rs.a + a * p.rs.b;
                if (NB <= PREFETCH_R_MAX_NB) {  // the old values were fetched before the k loop
                    *rd = (p.beta == 0.0) ? p.alpha * val : p.beta * rold[t][0] + p.alpha * val;
                    if (p.pair && a != b) *rm = (p.beta == 0.0) ? p.alpha * val : p.beta * rold[t][1] + p.alpha * val;
                } else {
                    r_update(rd, val, p.alpha, p.beta);
                    if (p.pair && a != b) r_update(rm, val, p.alpha, p.beta);
                }
            }
        }
    }
}

// Copies of L and t2 with padded rows (the pad columns are zero) and t2 in (i,j) order, for the bulk copies of k_small_fused:
// Lp[P][a][ld] (ld = nvirt rounded up to even), tp[i*o+j][c][ldt] (ldt = SmallCfg::LDT: conflict-free reads in step 1).  Either source may be null (no copy needed).
__global__ void __launch_bounds__(256) k_small_prepack(const double *__restrict__ L, const double *__restrict__ t2, double *__restrict__ Lp,
                                                      double *__restrict__ tp, int o, int v, int x, int ld, int ldt, RStrides ts) {
    const int64_t nL = L ? (int64_t)x * v * ld : 0, nT = t2 ? (int64_t)o * o * v * ldt : 0;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < nL + nT; idx += (int64_t)gridDim.x * blockDim.x) {
        if (idx < nL) {
            const int c = (int)(idx % ld);
            const int64_t row = idx / ld;  // P * v + a
            Lp[idx] = c < v ? __ldg(L + row * v + c) : 0.0;
        } else {
            const int64_t e = idx - nL;
            const int d = (int)(e % ldt);
            int64_t r = e / ldt;
            const int c = (int)(r % v);
            r /= v;
            const int j = (int)(r % o), i = (int)(r / o);
            tp[e] = d < v ? __ldg(t2 + i * ts.i + j * ts.j + c * ts.a + d) : 0.0;
        }
    }
}

}  // namespace ppl
