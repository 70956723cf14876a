// ppl_kernels_full.cuh -- kernels of PPL_SYM_FULL: the path with the full 8-fold ERI symmetry.
//
// Preconditions (both hold for real orbitals and CC amplitudes; north_star names both):
//   L[P,a,c] == L[P,c,a]   =>  X[ab][cd] := (ac|bd) is invariant under a<->c, b<->d, (ac)<->(bd)
//   t2[i,j,c,d] == t2[j,i,d,c]
// With the packed pair indices I = (a<=b), J = (c<=d) and
//   S+-[I][J] = (ac|bd) +- (ad|bc)                 (a SYMMETRIC matrix in (I,J), for + and for -)
//   tau+-[(i<=j)][J] = (t2[ij,cd] +- t2[ij,dc])/2  (J diagonal c==d: t2[ij,cc]/2, so that S+ needs no special case)
//   R+-[(i<=j)][I] = sum_J tau+-[.][J] S+-[I][J],  R[i,j,a,b] = R+ + R-,  R[j,i,a,b] = R+ - R-  (and the pair mirror)
// only the blocks of S+- on or above the diagonal are generated, each used twice.  The virtual index
// is cut into a-blocks A of 16; for slab A (all four indices >= A0, a in A):
//   step 0  (one launch per slab)  strip X[(a,b)][(c,d)], b,c,d >= A0: a GEMM over P with rows m = (c, a_l)
//           and columns n = (b, d) restricted to d-block >= b-block; the b<->d mirror image is stored too
//           (the a<->c image is what lets the rows be the 16 contiguous L[P][c][A0..A0+16) -- one TMA box)
//   fold    per tile (A; b-group): W+-[(a,b)][J], J >= (A0,A0); rows with a > b are written as zeros
//   use 1   R+-acc[.][(a,b)] += tau+-[.][J >= (A0,A0)] . W+-[(a,b)][J]^T     (k_step1_tma, split-K, k_reduce_acc)
//   use 2   R+-acc[.][J]     += tau+-[.][(a,b) in tile] . W+-[(a,b)][J],  J >= (A0+16, A0+16)   (k_step1t_tma)
// and one k_unpack_full at the end writes R.  Executed flops: step 0 ~ 1/8, step 1 ~ 1/4 of nominal.
// The identity is pinned on the CPU by tests/test_oracle_pins.py::test_full_symmetry_hook_identity.
#pragma once
#include "ppl_kernels_tma.cuh"

namespace ppl {


// ---------------------------------------------------------------------------------------------
// step 0 of one slab.  mapL as in k_step0_tma: {inner = nvirt^2, outer = nchol}, box {16, BK}.
// Row tile tm: 8 boxes, box i <-> c = A0 + 8 tm + i, inner coordinate c*v + A0 (16 a's of L[P][c][.]).
// Column tile tn: 8 boxes, box j <-> chunk 8 tn + j of the slab's chunk table: (b, d0) -> coordinate
// b*v + d0 (16 d's of L[P][b][.]); b < 0 marks padding.  Chunks of one b start at its own 16-block.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_pack_diag(const double *__restrict__ L, double *__restrict__ Lq, int x, int v, int nfull,
                                                  int64_t ldq) {
    const int64_t per_p = (int64_t)nfull * DIAG_PACKED, total = (int64_t)x * per_p;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t P = idx / per_p;
        const int r = (int)(idx - P * per_p), blk = r / DIAG_PACKED, t = r - blk * DIAG_PACKED;
        int bl, dl;
        double val = 0.0;
        if (diag_unpack(t, bl, dl)) val = __ldg(L + (P * v + 16 * blk + bl) * v + 16 * blk + dl);
        Lq[P * ldq + r] = val;
    }
}

struct Step0SlabArgs {
    int A0, ta;          // first a of the slab, number of a's (16 except in the last slab)
    int v, K;            // nvirt, nchol
    int tiles_m, tiles_n;
    const int2 *chunks;  // [8 * tiles_n] (b, d0)
    double *X;           // strip [(a_l * rows_per_a + b - b_base)][c * v + d], row stride v*v
    int rows_per_a;      // strip rows per a_l: v (the slab's whole strip) or the b-group width (memory-tight mode)
    int b_base;          // first b of the strip: 0, or the b-group's first b
    int group_m;         // raster: row tiles per group (12: a wave of 148 CTAs covers ~12 x 12 tiles, the fewest operand panels per
                         // wave; taller groups read MORE from DRAM -- measured, profiles/r02_step0_l2.md)
    int hints;           // L2 policy bits (ppl_debug_opts_t.full_hints): 1 evict_last row panels, 2 evict_first column panels, 4 streaming stores
    int image;           // 1: chunks cover d-block >= b-block only and the epilogue stores the b<->d image too (rows of
                         // every b >= A0 must be in the strip); 0: the chunks cover the full (b, d) rectangle of the group
};

__global__ void __launch_bounds__(TMA_THREADS, 1)
    k_step0_slab(const __grid_constant__ CUtensorMap mapL, const __grid_constant__ CUtensorMap mapQ, const Step0SlabArgs p) {
    extern __shared__ unsigned char smem_raw[];
    const TmaSmem sm = carve_smem(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    init_barriers(sm, tid);

    const int num_items = p.tiles_m * p.tiles_n;
    const int nkt = (p.K + BK - 1) / BK;
    const int v = p.v, vv = v * v;

    if (warp >= CONSUMER_WARPS) {
        setmaxnreg_dec<PRODUCER_REGS>();
        if (warp == CONSUMER_WARPS && lane == 0) {
            prefetch_tmap(&mapL);
            prefetch_tmap(&mapQ);
            int stage = 0;
            uint32_t phase = 0;
            for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
                int tm, tn;
                raster(item, p.tiles_m, p.tiles_n, tm, tn, p.group_m);
                int xa[8], xb[8];
                unsigned packed = 0;  // bit i: chunk i of the column tile comes from the packed diagonal blocks (mapQ)
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int c = p.A0 + 8 * tm + i;
                    xa[i] = c < v ? c * v + p.A0 : vv;  // beyond the tensor: the box is zero-filled
                    const int2 ch = p.chunks[8 * tn + i];
                    xb[i] = ch.x >= 0 ? ch.x * v + ch.y : (ch.x == -1 ? vv : ch.y);
                    packed |= (ch.x <= -2 ? 1u : 0u) << i;
                }
                const uint64_t pol_a = (p.hints & 1) ? L2_EVICT_LAST : L2_EVICT_NORMAL, pol_b = (p.hints & 2) ? L2_EVICT_FIRST : L2_EVICT_NORMAL;
                for (int kt = 0; kt < nkt; ++kt) {
                    mbar_wait(&sm.empty[stage], phase ^ 1);
                    mbar_expect_tx(&sm.full[stage], STAGE_BYTES);
                    double *da = sm.a + (size_t)stage * BM * BK, *db = sm.b + (size_t)stage * BN * BK;
#pragma unroll
                    for (int i = 0; i < 8; ++i) tma_load_2d_hint(da + i * BK * 16, &mapL, xa[i], kt * BK, &sm.full[stage], pol_a);
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        tma_load_2d_hint(db + i * BK * 16, ((packed >> i) & 1) ? &mapQ : &mapL, xb[i], kt * BK, &sm.full[stage], pol_b);
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
    const int offk_even = q * 16 + ((c ^ q) << 1);
    const int offk_odd = (q + 4) * 16 + ((c ^ (q + 4)) << 1);
    int stage = 0, rel_stage = -1;
    uint32_t phase = 0;
    for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
        int tm, tn;
        raster(item, p.tiles_m, p.tiles_n, tm, tn, p.group_m);
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
            rel_stage = stage;
            if (++stage == TSTAGES) {
                stage = 0;
                phase ^= 1;
            }
        }
        // epilogue.  block (2i+e, 2j+f): row m = 64 wm + 16 i + 2c(g) + e  <->  c = A0 + 8 tm + 4 wm + i, a_l = 2c(g) + e
        //            col  n = 32 wn + 16 j + 2q + 8h + f                  <->  chunk 8 tn + 2 wn + j, d = d0 + 2q + 8h + f
        int2 ch[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) ch[j] = p.chunks[8 * tn + 2 * wn + j];
        // the chunk table is d-block major with b ascending: a thread's two chunks are normally (b, d0), (b+1, d0) with b
        // even, and then the b<->d image of both is ONE 16-byte store per d (X[a,d,c,b..b+1])
        const bool pair = ch[0].x >= 0 && ch[1].x == ch[0].x + 1 && ch[1].y == ch[0].y && (ch[0].x & 1) == 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int cc = p.A0 + 8 * tm + 4 * wm + i;
            if (cc >= v) continue;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int al = 2 * c + e;
                if (al >= p.ta) continue;
                double *xa = p.X + ((int64_t)al * p.rows_per_a - p.b_base) * vv + (int64_t)cc * v;  // + b*vv + d
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int b = ch[j].x, d0 = ch[j].y;
                    if (b == -1) continue;
                    if (b <= -2) {  // packed diagonal block: column t of the triangle -> (b_l <= d_l), plus the b<->d image
                        const int blk = -2 - b, t0 = d0 - blk * DIAG_PACKED + 2 * q;
#pragma unroll
                        for (int h = 0; h < 2; ++h)
#pragma unroll
                            for (int f = 0; f < 2; ++f) {
                                int bl, dl;
                                if (!diag_unpack(t0 + 8 * h + f, bl, dl)) continue;
                                const double val = acc[2 * i + e][2 * j + f][h];
                                const int bb = 16 * blk + bl, dd = 16 * blk + dl;
                                xa[(int64_t)bb * vv + dd] = val;
                                if (bl != dl) xa[(int64_t)dd * vv + bb] = val;
                            }
                        continue;
                    }
                    const bool offdiag = p.image && d0 != p.A0 + ((b - p.A0) & ~15);  // d-block above the b-block: store the b<->d image too
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int d = d0 + 2 * q + 8 * h;
                        const double v0 = acc[2 * i + e][2 * j][h], v1 = acc[2 * i + e][2 * j + 1][h];
                        if (d + 1 < v) {  // v even (TMA path), d even: 16-byte aligned
                            if (p.hints & 4)
                                __stcs(reinterpret_cast<double2 *>(xa + (int64_t)b * vv + d), make_double2(v0, v1));
                            else
                                *reinterpret_cast<double2 *>(xa + (int64_t)b * vv + d) = make_double2(v0, v1);
                            if (offdiag && !pair) {
                                xa[(int64_t)d * vv + b] = v0;
                                xa[(int64_t)(d + 1) * vv + b] = v1;
                            }
                        } else if (d < v) {
                            xa[(int64_t)b * vv + d] = v0;
                            if (offdiag && !pair) xa[(int64_t)d * vv + b] = v0;
                        }
                    }
                }
                if (pair && p.image) {
                    const int b = ch[0].x, d0 = ch[0].y;
                    if (d0 != p.A0 + ((b - p.A0) & ~15)) {  // b, b+1 share a 16-block (b even)
#pragma unroll
                        for (int h = 0; h < 2; ++h)
#pragma unroll
                            for (int f = 0; f < 2; ++f) {
                                const int d = d0 + 2 * q + 8 * h + f;
                                if (d < v)
                                    *reinterpret_cast<double2 *>(xa + (int64_t)d * vv + b) =
                                        make_double2(acc[2 * i + e][f][h], acc[2 * i + e][2 + f][h]);
                            }
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// use 2:  acc[m][n] += sum_r tau[m][kappa(r)] W[r][n],   n in [n_begin, n_end)
// r = 16 kt + t runs over the rows (a_l, b_l) of the W tile: kt <-> (a = A0 + kt / kt_per_a, sixteen b's from
// b1 = bg0 + 16 (kt % kt_per_a)), whose packed indices kappa = kplus(a, b1) + t (kminus for the - part) are
// CONTIGUOUS in tau and start 16-byte aligned (ppl_kernels.cuh, kplus): one TMA box per k-tile.  Positions with b < a, b >= v or a beyond the slab address other
// (finite) entries of tau or fall outside the tensor (zero fill); the fold wrote those rows of W as zeros.
// mapA: tau as {inner = Kp, outer = M}, box {16, 16 NI} (the map of use 1).  mapB: the W slot as
// {inner = Kp, outer = rows}, box {16, 16}: operand tile 16 (k) x 128 (n) as 8 boxes, n contiguous.
// ---------------------------------------------------------------------------------------------
struct Step1TArgs {
    int M;
    int range;           // 1: the W rows are a run of the packed pair index: k-tile kt <-> tau columns kap0 + 16 kt (kt_per_a, A0, bg0 unused)
    int kap0;
    int n_base;          // n_begin rounded down to a multiple of 16: the column of tile 0
    int n_begin, n_end;
    int nkt, kt_per_a;
    int A0, bg0, v;
    int minus;
    MSplit ms;           // row tiling of M (ppl_kernels_tma.cuh)
    double *acc;         // [M][ld]
    int64_t ld;
};

// k loop of one work item of use 2 for a warp that owns NA 8-row blocks (see step1_consume)
template <int NI, int NA>
__device__ __forceinline__ void step1t_consume(double (&acc)[NI][2][2][2], const TmaSmem &sm, int as_off, int bs_off, int offa0, int offa1,
                                               int offb_e0, int offb_e1, int nkt, int nact, int &stage, uint32_t &phase, int &rel_stage,
                                               int lane) {
    constexpr int BM1 = Step1Cfg<NI>::BM1;
    for (int kt = 0; kt < nkt; ++kt) {
        mbar_wait(&sm.full[stage], phase);
        release_previous(sm, rel_stage, lane);
        const double *as = sm.a + (size_t)stage * BM1 * BK + as_off;
        const double *bs = sm.b + (size_t)stage * BN * BK + bs_off;
#pragma unroll
        for (int k8 = 0; k8 < BK / 8; ++k8) {
            double2 a[NA > 0 ? NA : 1], b0[2], b1[2];
#pragma unroll
            for (int i = 0; i < NA; ++i)
                a[i] = *reinterpret_cast<const double2 *>(as + i * 8 * BK + (k8 ? offa1 : offa0));
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                b0[j] = *reinterpret_cast<const double2 *>(bs + j * (BK * 16) + k8 * 128 + offb_e0);
                b1[j] = *reinterpret_cast<const double2 *>(bs + j * (BK * 16) + k8 * 128 + offb_e1);
            }
#pragma unroll
            for (int i = 0; i < NA; ++i)
                {
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        dmma(acc[i][j][0][0], acc[i][j][0][1], a[i].x, b0[j].x);
                        dmma(acc[i][j][1][0], acc[i][j][1][1], a[i].x, b0[j].y);
                    }
                }
#pragma unroll
            for (int i = 0; i < NA; ++i)
                {
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        dmma(acc[i][j][0][0], acc[i][j][0][1], a[i].y, b1[j].x);
                        dmma(acc[i][j][1][0], acc[i][j][1][1], a[i].y, b1[j].y);
                    }
                }
        }
        rel_stage = stage;
        if (++stage == TSTAGES) {
            stage = 0;
            phase ^= 1;
        }
    }
}

template <int NI>
__global__ void __launch_bounds__(TMA_THREADS, 1)
    k_step1t_tma(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const Step1TArgs p) {
    using Cfg = Step1Cfg<NI>;
    constexpr int BM1 = Cfg::BM1;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    unsigned char *al = smem_raw + ((1024u - (base & 1023u)) & 1023u);
    TmaSmem sm;
    sm.a = reinterpret_cast<double *>(al);
    sm.b = reinterpret_cast<double *>(al + (size_t)TSTAGES * Cfg::A_BYTES);
    sm.full = reinterpret_cast<uint64_t *>(al + (size_t)TSTAGES * Cfg::STAGE);
    sm.empty = sm.full + TSTAGES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    init_barriers(sm, tid);

    const int tiles_m = p.ms.tiles_m, tiles_n = (p.n_end - p.n_base + BN - 1) / BN;
    const int num_items = tiles_m * tiles_n;

    if (warp >= CONSUMER_WARPS) {
        setmaxnreg_dec<PRODUCER_REGS>();
        if (warp == CONSUMER_WARPS && lane == 0) {
            prefetch_tmap(&mapA);
            prefetch_tmap(&mapB);
            int stage = 0;
            uint32_t phase = 0;
            for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
                const int tm = item % tiles_m, tn = item / tiles_m;
                const int n0 = p.n_base + tn * BN;
                int row0, ni0, ni1;
                m_tile(p.ms, tm, row0, ni0, ni1);
                for (int kt = 0; kt < p.nkt; ++kt) {
                    int64_t kap;
                    if (p.range) {
                        kap = (int64_t)p.kap0 + 16 * kt;  // even: the run starts at an even index
                    } else {
                        const int a = p.A0 + kt / p.kt_per_a, b1 = p.bg0 + 16 * (kt % p.kt_per_a);
                        kap = p.minus ? kminus(a, b1, p.v) : kplus(a, b1, p.v);  // even: b1 is a multiple of 16
                    }
                    mbar_wait(&sm.empty[stage], phase ^ 1);
                    mbar_expect_tx(&sm.full[stage], Cfg::STAGE);
                    tma_load_2d(sm.a + (size_t)stage * BM1 * BK, &mapA, (int)kap, row0, &sm.full[stage]);
                    double *db = sm.b + (size_t)stage * BN * BK;
#pragma unroll
                    for (int i = 0; i < 8; ++i) tma_load_2d(db + i * BK * 16, &mapB, n0 + 16 * i, kt * BK, &sm.full[stage]);
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
    // A (k contiguous): row 8i + c, 16-byte chunk (4 k8 + q) ^ c  ->  k = 8 k8 + 2q, 2q + 1
    const int offa0 = c * 16 + ((q ^ c) << 1);
    const int offa1 = c * 16 + (((4 + q) ^ c) << 1);
    // B (n contiguous): box j2 of the warp's two, row rho = 8 k8 + 2q + e, chunk g ^ (rho & 7)  ->  n = 16 j2 + 2g, 2g + 1
    const int offb_e0 = (2 * q) * 16 + ((g ^ (2 * q)) << 1);
    const int offb_e1 = (2 * q + 1) * 16 + ((g ^ (2 * q + 1)) << 1);
    int stage = 0, rel_stage = -1;
    uint32_t phase = 0;
    for (int item = blockIdx.x; item < num_items; item += gridDim.x) {
        const int tm = item % tiles_m;
        int row0, ni0, ni1;
        m_tile(p.ms, tm, row0, ni0, ni1);
        const int nact = wm ? ni1 : ni0;
        const int wrow = wm ? 8 * ni0 : 0;
        // acc[i][j2][f][h]: row m = 8i + c(g); h = 0 <-> n = 16 j2 + 4q + f, h = 1 <-> n = 16 j2 + 4q + 2 + f
        double acc[NI][2][2][2];
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) acc[i][j][0][0] = acc[i][j][0][1] = acc[i][j][1][0] = acc[i][j][1][1] = 0.0;

        if (nact == NI)
            step1t_consume<NI, NI>(acc, sm, wrow * BK, (wn * 2) * (BK * 16), offa0, offa1, offb_e0, offb_e1, p.nkt, nact, stage,
                                          phase, rel_stage, lane);
        else  // nact == NI - 1: the host's row tiling hands a warp NI or NI - 1 blocks, nothing else (m_geom_tma)
            step1t_consume<NI, NI - 1>(acc, sm, wrow * BK, (wn * 2) * (BK * 16), offa0, offa1, offb_e0, offb_e1, p.nkt, nact,
                                              stage, phase, rel_stage, lane);
        // epilogue: accumulate into the R+- matrix.  Every element belongs to exactly one item of this launch and
        // launches are ordered on the stream, so the sequence of additions per element is fixed (bit-reproducible);
        // the adds are issued as reductions (RED.ADD.F64, no return value): no load latency in the epilogue.
        int it2 = item;  // tile coordinates derived again behind an opaque move: nothing of them stays live across the k loop
        asm volatile("" : "+r"(it2));
        int erow0, eni0, eni1;
        m_tile(p.ms, it2 % tiles_m, erow0, eni0, eni1);
        const int enact = wm ? eni1 : eni0, en0 = p.n_base + (it2 / tiles_m) * BN;
        erow0 += wm ? 8 * eni0 : 0;
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const int m = erow0 + 8 * i + c;
            if (i >= enact || m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int n = en0 + wn * WTN + 16 * j + 4 * q;  // multiple of 4; rows are 128-byte aligned
                double *dst = p.acc + (int64_t)m * p.ld + n;
                const double vals[4] = {acc[i][j][0][0], acc[i][j][1][0], acc[i][j][0][1], acc[i][j][1][1]};
#pragma unroll
                for (int t = 0; t < 4; ++t)
                    if (n + t >= p.n_begin && n + t < p.n_end) atomicAdd(dst + t, vals[t]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// use 1 reduction: Racc[m][kidx(a,b)] += sum_z part[z][m][n], n = a_l*tbp + b_l, for a <= b (plus) / a < b (minus)
// ---------------------------------------------------------------------------------------------
struct ReduceAccArgs {
    const double *part;  // [splitk][M][N]
    int splitk, M, N;
    int tbp, A0, ta, bg0, v;
    int minus;
    double *acc;
    int64_t ld;
};

__global__ void __launch_bounds__(256) k_reduce_acc(const ReduceAccArgs p) {
    const int64_t MN = (int64_t)p.M * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < MN; idx += (int64_t)gridDim.x * blockDim.x) {
        const int m = (int)(idx / p.N), n = (int)(idx - (int64_t)m * p.N);
        const int al = n / p.tbp, bl = n - al * p.tbp;
        const int a = p.A0 + al, b = p.bg0 + bl;
        if (al >= p.ta || b >= p.v || a > b || (p.minus && a == b)) continue;
        double s = 0.0;
        for (int z = 0; z < p.splitk; ++z) s += p.part[(int64_t)z * MN + idx];
        const int64_t k = p.minus ? kminus(a, b, p.v) : kplus(a, b, p.v);
        p.acc[(int64_t)m * p.ld + k] += s;
    }
}

// the same for W+- rows that are a run of the packed pair index: Racc[m][k0 + n] += sum_z part[z][m][n] (holes of the
// packed layout are rows of zeros in W+-, so they receive += 0)
struct ReduceRangeArgs {
    const double *part;  // [splitk][M][N]
    int splitk, M, N;
    int k0;
    double *acc;
    int64_t ld;
};
__global__ void __launch_bounds__(256) k_reduce_range(const ReduceRangeArgs p) {
    const int64_t MN = (int64_t)p.M * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < MN; idx += (int64_t)gridDim.x * blockDim.x) {
        const int m = (int)(idx / p.N), n = (int)(idx - (int64_t)m * p.N);
        double s = 0.0;
        for (int z = 0; z < p.splitk; ++z) s += p.part[(int64_t)z * MN + idx];
        p.acc[(int64_t)m * p.ld + p.k0 + n] += s;
    }
}

// ---------------------------------------------------------------------------------------------
// final unpack: R[i,j,a,b] = beta R + alpha (R+[(ij)][(ab)] + s R-[(ij)][(ab)]), s = +1 if (i,j) and (a,b) are
// both in order or both swapped, -1 otherwise; R- = 0 on i == j or a == b.  One thread per R element.
// ---------------------------------------------------------------------------------------------
struct UnpackArgs {
    const double *rp, *rm;
    int64_t ldp, ldm;
    int o, v;            // v: the caller's nvirt (extent of a, b in R)
    int vk;              // nvirt of the packed geometry (v rounded up to even)
    double alpha, beta;
    RStrides rs;
    double *R;           // base of the array the strides address, after r_bias elements are subtracted from the offset
    int64_t r_bias = 0;  // 0: the caller's R; a slab buffer holding the a's [a0, a0 + na) passes its own base and a0 * rs.a
    int64_t idx0, idx1;  // range of the flattened (i,j,a_l,b) index that is written (all: 0, o^2 na v)
    int a0, na;          // the a's covered: a = a0 + a_l, a_l < na (all: 0, v).  A slab of a's is complete as soon as its own slab
                         // of the PPL_SYM_FULL loop is: ppl_apply_host unpacks and ships R[:, :, slab, :] while later slabs run
};

__global__ void __launch_bounds__(256) k_unpack_full(const UnpackArgs p) {
    for (int64_t idx = p.idx0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < p.idx1; idx += (int64_t)gridDim.x * blockDim.x) {
        const int b = (int)(idx % p.v);
        int64_t r = idx / p.v;
        const int a = p.a0 + (int)(r % p.na);
        r /= p.na;
        const int j = (int)(r % p.o), i = (int)(r / p.o);
        const int i1 = min(i, j), j1 = max(i, j), a1 = min(a, b), b1 = max(a, b);
        double val = p.rp[rowplus(i1, j1, p.o) * p.ldp + kplus(a1, b1, p.vk)];
        if (i1 != j1 && a1 != b1) {
            const double rm = p.rm[rowminus(i1, j1, p.o) * p.ldm + kminus(a1, b1, p.vk)];
            val += ((i > j) == (a > b)) ? rm : -rm;
        }
        r_update(p.R + (i * p.rs.i + j * p.rs.j + a * p.rs.a + b * p.rs.b - p.r_bias), val, p.alpha, p.beta);
    }
}

// ---------------------------------------------------------------------------------------------
// odd nvirt: L[x][v][v] -> Lpad[x][vp][vp], vp = v + 1, the pad row and column zero.  Rows of Lpad are 16-byte
// aligned (TMA-legal) and the pad index contributes exact zeros everywhere downstream.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_pad_L(const double *__restrict__ L, double *__restrict__ Lpad, int x, int v, int vp) {
    const int64_t total = (int64_t)x * vp * vp;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(idx % vp);
        const int64_t r = idx / vp;
        const int a = (int)(r % vp);
        const int64_t P = r / vp;
        Lpad[idx] = (a < v && c < v) ? __ldg(L + (P * v + a) * v + c) : 0.0;
    }
}

}  // namespace ppl
