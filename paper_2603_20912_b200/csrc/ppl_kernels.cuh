// ppl_kernels.cuh -- sm_100a kernels of the pp-ladder path (FP64, DMMA m8n8k4).
//
// step 0  (PAPER.md:118-120 'xac,xbd->acbd', eq. 5 l.63):  W[(a,b)][(c,d)] = sum_P L[P,a,c] L[P,b,d]
// step 1  (PAPER.md:118-120 'acbd,ecfd->efab', eq. 4/6):   part[z][(i,j)][(a,b)] = sum_{(c,d) in chunk z} t2[(i,j)][(c,d)] W[(a,b)][(c,d)]
// reduce  ("add to view of final result"):    R[i,j,a,b] += sum_z part[z]; mirror R[j,i,b,a] += same
//
// Both GEMMs run on the FP64 tensor pipe (SASS DMMA.8x8x4): measured 37.1 TFLOP/s on B200 against
// 33.9 for DFMA, with no gain from mixing the two (same pipe) -- see DESIGN.md.  tcgen05/TMEM has
// no FP64 kind, so accumulators live in registers; operands are staged global->shared with
// cp.async (16-byte when rows are 16-byte aligned, else 8-byte) through a STAGES-deep ring.
//
// Fragment layout of mma.sync.aligned.m8n8k4.row.col.f64 (verified on the device by
// tests/test_gpu_parity.py::test_dmma_fragment_layout): lane = 4*g + q,
//   A(8x4): a = A[g][q]      B(4x8): b = B[q][g]      C(8x8): c0 = C[g][2q], c1 = C[g][2q+1].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppl_device.cuh"

namespace ppl {

// ---------------------------------------------------------------------------------------------
// step 0: both operands MN-contiguous ("k-outer"): A[k][m] = L[P=k][a0 + m/v][m%v], B likewise.
// ---------------------------------------------------------------------------------------------
struct Step0Args {
    const double *A;  // L + a0*v      (row k at A + k*ld)
    const double *B;  // L + b0*v
    int64_t ld;       // v*v
    int M, N, K;      // ta*v, tb*v, nchol
    int v, tb;        // nvirt; number of b in this tile
    double *W;        // tile [ta*tb][ldw], row (a_l*tb + b_l), col c*v + d
    int64_t ldw;
};

template <int VEC>  // doubles per async copy: 2 (16 B) or 1 (8 B)
__device__ __forceinline__ void load_mn(double *s, const double *g, int64_t ld, int k0, int Kend, int x0, int X, int tid) {
    // tile BK rows (k) x BM cols (contiguous x); s is [BK][LDS_MN]
    constexpr int CPR = BM / VEC;  // chunks per row
#pragma unroll
    for (int c = 0; c < (BK * CPR) / NTHREADS; ++c) {
        const int idx = tid + c * NTHREADS;
        const int row = idx / CPR, ch = idx % CPR;
        const int k = k0 + row, x = x0 + ch * VEC;
        int nb = (k < Kend) ? (X - x) * 8 : 0;
        nb = max(0, min(nb, VEC * 8));
        const double *src = nb > 0 ? g + (int64_t)k * ld + x : g;
        if (VEC == 2)
            cp_async16(s + row * LDS_MN + ch * VEC, src, nb);
        else
            cp_async8(s + row * LDS_MN + ch * VEC, src, nb);
    }
}

template <int VEC>
__global__ void __launch_bounds__(NTHREADS, 1) k_step0(const Step0Args p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *As = reinterpret_cast<double *>(smem_raw);
    double *Bs = As + STAGES * BK * LDS_MN;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    const int tiles_m = (p.M + BM - 1) / BM, tiles_n = (p.N + BN - 1) / BN;
    int tm, tn;
    raster(blockIdx.x, tiles_m, tiles_n, tm, tn);
    const int m0 = tm * BM, n0 = tn * BN;
    const int nkt = (p.K + BK - 1) / BK;

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) {
            load_mn<VEC>(As + s * BK * LDS_MN, p.A, p.ld, s * BK, p.K, m0, p.M, tid);
            load_mn<VEC>(Bs + s * BK * LDS_MN, p.B, p.ld, s * BK, p.K, n0, p.N, tid);
        }
        cp_async_commit();
    }
    for (int kt = 0; kt < nkt; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int kn = kt + STAGES - 1;
            if (kn < nkt) {
                const int s = kn % STAGES;
                load_mn<VEC>(As + s * BK * LDS_MN, p.A, p.ld, kn * BK, p.K, m0, p.M, tid);
                load_mn<VEC>(Bs + s * BK * LDS_MN, p.B, p.ld, kn * BK, p.K, n0, p.N, tid);
            }
            cp_async_commit();
        }
        const double *as = As + (kt % STAGES) * BK * LDS_MN + wm * WTM + 2 * g;
        const double *bs = Bs + (kt % STAGES) * BK * LDS_MN + wn * WTN + 2 * g;
#pragma unroll
        for (int k4 = 0; k4 < BK / 4; ++k4) {
            const int row = k4 * 4 + q;
            double2 a[4], b[2];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = *reinterpret_cast<const double2 *>(as + row * LDS_MN + 16 * i);
#pragma unroll
            for (int j = 0; j < 2; ++j) b[j] = *reinterpret_cast<const double2 *>(bs + row * LDS_MN + 16 * j);
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
    }
    cp_async_wait<0>();

    // epilogue: accumulator block (2i+e, 2j+f): row g <-> m = mw + 16i + 2g + e,
    //           cols 2q,2q+1 <-> n = nw + 16j + 4q + f and nw + 16j + 4q + 2 + f.
    const int v = p.v;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int m = m0 + wm * WTM + 16 * i + 2 * g + e;
            if (m >= p.M) continue;
            const int al = m / v, c = m - al * v;
            double *wrow = p.W + (int64_t)al * p.tb * p.ldw + (int64_t)c * v;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int nb = n0 + wn * WTN + 16 * j + 4 * q;
                const double vals[4] = {acc[2 * i + e][2 * j][0], acc[2 * i + e][2 * j + 1][0],
                                        acc[2 * i + e][2 * j][1], acc[2 * i + e][2 * j + 1][1]};
                const int bl = nb / v, d = nb - bl * v;
                if ((v & 3) == 0 && nb + 3 < p.N) {  // 4 consecutive n stay inside one b and are 32-B aligned
                    double *dst = wrow + (int64_t)bl * p.ldw + d;
                    *reinterpret_cast<double2 *>(dst) = make_double2(vals[0], vals[1]);
                    *reinterpret_cast<double2 *>(dst + 2) = make_double2(vals[2], vals[3]);
                } else {
#pragma unroll
                    for (int t = 0; t < 4; ++t) {
                        const int n = nb + t;
                        if (n < p.N) {
                            const int bl2 = n / v, d2 = n - bl2 * v;
                            wrow[(int64_t)bl2 * p.ldw + d2] = vals[t];
                        }
                    }
                }
            }
        }
}

// ---------------------------------------------------------------------------------------------
// step 1: both operands K-contiguous: A[m][k] = t2[(i,j)=m][(c,d)=k], B[n][k] = W[(a,b)=n][(c,d)=k].
// smem rows are BK=16 doubles = 8 chunks of 16 B; chunk index XOR ((row&1)<<2) makes the
// 128-bit fragment loads (rows g, chunks q) bank-conflict-free without padding.
// ---------------------------------------------------------------------------------------------
struct Step1Args {
    const double *A;  // t2
    const double *B;  // W tile
    int64_t lda, ldb; // v*v, ldw
    int M, N, K;      // nocc^2, ta*tb, nvirt^2
    int k_per_split;  // multiple of BK
    double *part;     // [splitk][M][N]
};

template <int VEC>
__device__ __forceinline__ void load_k(double *s, const double *g, int64_t ld, int k0, int Kend, int x0, int X, int tid) {
    // tile BM rows (x) x BK cols (contiguous k); s is [BM][BK] swizzled
    constexpr int CPR = BK / VEC;
#pragma unroll
    for (int c = 0; c < (BM * CPR) / NTHREADS; ++c) {
        const int idx = tid + c * NTHREADS;
        const int row = idx / CPR, ch = idx % CPR;
        const int x = x0 + row, k = k0 + ch * VEC;
        int nb = (x < X) ? (Kend - k) * 8 : 0;
        nb = max(0, min(nb, VEC * 8));
        const double *src = nb > 0 ? g + (int64_t)x * ld + k : g;
        if (VEC == 2) {
            cp_async16(s + row * BK + ((ch ^ ((row & 1) << 2)) << 1), src, nb);
        } else {
            cp_async8(s + row * BK + ((((ch >> 1) ^ ((row & 1) << 2)) << 1) | (ch & 1)), src, nb);
        }
    }
}

template <int VEC>
__global__ void __launch_bounds__(NTHREADS, 1) k_step1(const Step1Args p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *As = reinterpret_cast<double *>(smem_raw);
    double *Bs = As + STAGES * BM * BK;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    const int tiles_m = (p.M + BM - 1) / BM;
    const int tm = blockIdx.x % tiles_m, tn = blockIdx.x / tiles_m;
    const int m0 = tm * BM, n0 = tn * BN;
    const int z = blockIdx.y;
    const int Kbeg = z * p.k_per_split;
    const int Kend = min(p.K, Kbeg + p.k_per_split);
    const int nkt = max(0, (Kend - Kbeg + BK - 1) / BK);

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) {
            load_k<VEC>(As + s * BM * BK, p.A, p.lda, Kbeg + s * BK, Kend, m0, p.M, tid);
            load_k<VEC>(Bs + s * BN * BK, p.B, p.ldb, Kbeg + s * BK, Kend, n0, p.N, tid);
        }
        cp_async_commit();
    }
    const int swz = (g & 1) << 2;
    for (int kt = 0; kt < nkt; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int kn = kt + STAGES - 1;
            if (kn < nkt) {
                const int s = kn % STAGES;
                load_k<VEC>(As + s * BM * BK, p.A, p.lda, Kbeg + kn * BK, Kend, m0, p.M, tid);
                load_k<VEC>(Bs + s * BN * BK, p.B, p.ldb, Kbeg + kn * BK, Kend, n0, p.N, tid);
            }
            cp_async_commit();
        }
        const double *as = As + (kt % STAGES) * BM * BK + (wm * WTM + g) * BK;
        const double *bs = Bs + (kt % STAGES) * BN * BK + (wn * WTN + g) * BK;
#pragma unroll
        for (int k8 = 0; k8 < BK / 8; ++k8) {
            const int off = ((k8 * 4 + q) ^ swz) << 1;
            double2 a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = *reinterpret_cast<const double2 *>(as + i * 8 * BK + off);
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = *reinterpret_cast<const double2 *>(bs + j * 8 * BK + off);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
        }
    }
    cp_async_wait<0>();

    // epilogue: block (i,j): row g <-> m = mw + 8i + g; cols n = nw + 8j + 2q, +1
    double *part = p.part + (int64_t)z * p.M * p.N;
    const bool vec_ok = (p.N & 1) == 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int m = m0 + wm * WTM + 8 * i + g;
        if (m >= p.M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + wn * WTN + 8 * j + 2 * q;
            double *dst = part + (int64_t)m * p.N + n;
            if (vec_ok && n + 1 < p.N) {
                *reinterpret_cast<double2 *>(dst) = make_double2(acc[i][j][0], acc[i][j][1]);
            } else {
                if (n < p.N) dst[0] = acc[i][j][0];
                if (n + 1 < p.N) dst[1] = acc[i][j][1];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// reduce + accumulate + mirror (fixed summation order over z: bit-reproducible)
//   R = beta*R + alpha*sum_z part[z]   (beta == 0: overwrite, R is not read)
// R is addressed through four element strides so that both storage orders of SURVEY 8(f) NEXT-1
// ('ijab' = BASELINE.json / the paper's 'efab', and 'iajb' = the paper's 'iajb') are
// written in place -- the paper's transpose step folds into this addressing.
// Every R entry is touched exactly once per apply (tiles partition (a,b); the mirror covers the
// other triangle), so beta scaling here is exact.
// ---------------------------------------------------------------------------------------------
struct ReduceArgs {
    const double *part;  // [splitk][M][N]
    int splitk;
    int M, N;            // nocc^2, rows of this W tile
    int o, v, tb;        // nocc, nvirt, b count of this tile
    int a0, b0;          // first virtual index of the a / b block
    int n_off;           // row offset added to n before the (a,b) decode (dense-ERI slabs)
    int mirror;          // 1: also write R[j,i,b,a]
    double alpha, beta;
    RStrides rs;
    double *R;           // base of the array the strides address ...
    int64_t r_bias = 0;  // ... after this many elements are subtracted from the offset: 0 for the caller's R; a slab buffer that
                         // holds only the a's from a0 on passes its own base and a0 * rs.a (no pointer is formed outside it)
};

__global__ void __launch_bounds__(256) k_reduce(const ReduceArgs p) {
    const int64_t MN = (int64_t)p.M * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < MN; idx += (int64_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int z = 0; z < p.splitk; ++z) s += p.part[(int64_t)z * MN + idx];
        const int m = (int)(idx / p.N), n = (int)(idx - (int64_t)m * p.N) + p.n_off;
        const int al = n / p.tb, bl = n - al * p.tb;
        const int a = p.a0 + al, b = p.b0 + bl;
        const int i = m / p.o, j = m - i * p.o;
        r_update(p.R + (i * p.rs.i + j * p.rs.j + a * p.rs.a + b * p.rs.b - p.r_bias), s, p.alpha, p.beta);
        if (p.mirror) r_update(p.R + (j * p.rs.i + i * p.rs.j + b * p.rs.a + a * p.rs.b - p.r_bias), s, p.alpha, p.beta);
    }
}

// ---------------------------------------------------------------------------------------------
// PPL_SYM_PAIR_SA: symmetric / antisymmetric packing.
// For pair-symmetric t2 and ANY L, with (c,d) packed over c <= d (k+) and c < d (k-):
//   W+-[(ab)][k]  = X[(ab)][c,d] +- X[(ab)][d,c]          (X = step-0 tile (ac|bd); W+ diag = X[c,c])
//   tau+-[(ij)][k] = (t2[ij][c,d] +- t2[ij][d,c]) / 2      (i <= j rows only;   tau+ diag = t2[c,c])
//   R+- = tau+- W+-^T ;  R[i,j,a,b] = R+ + R- ;  R[j,i,a,b] = R+ - R-
// Both packings are the same gather: k_symfold does either (scale 1 for W, 1/2 for tau).
// ---------------------------------------------------------------------------------------------
struct FoldArgs {
    const double *src;   // row r, element (c,d) at src + roff(r) + c*sc + d   (d contiguous)
    int64_t sc;          // stride of c
    int64_t s_row;       // mode 0: row r at r*s_row;  mode 2: row (a_l, b) at (a_l*v + b)*s_row
    int64_t s_i, s_j;    // mode 1: row (i,j) at i*s_i + j*s_j - roff_bias
    int64_t roff_bias = 0;  // mode 1: elements in front of src that the array would have (a staged chunk of rows passes its own base)
    int mode;            // 0: fold W tile rows (every row has + and -); 1: pack amplitudes, rows (i<=j) of an o x o grid; 3: see below;
                         // 2: PPL_SYM_FULL: rows r = a_l*tbp + b_l of the tile (A; b-group) taken from the slab's strip;
                         //    rows with a > b, b >= v or a_l >= ta are written as zeros; only c >= A0 is touched
    int rows;            // mode 0/2: number of rows; mode 1: o*o (rows with i > j are skipped)
    int row0;            // first row processed (0 except when amplitudes are packed chunk by chunk: rows [row0, rows))
    int o, v;            // v: nvirt of the PACKED geometry (kplus/kminus, block grid): the caller's nvirt rounded up to even
    int vs;              // nvirt of the source: entries with c >= vs or d >= vs are read as zeros (the pad index of odd nvirt)
    double scale;        // factor of the off-diagonal (c<d) entries: 1 (W) or 1/2 (tau)
    double diag;         // factor of the diagonal (c==d) entries of the + part: PPL_SYM_PAIR_SA 1 (W), 1 (tau);
                         // PPL_SYM_FULL 2 (W), 1/2 (tau) -- same products, but W+ becomes a symmetric matrix
    int tbp, bg0, A0, ta;  // mode 2 (A0, ta also mode 3)
    int rows_per_a = 0, b_base = 0;  // mode 2/3: strip row of (a_l, b) is a_l * rows_per_a + b - b_base (v, 0: the slab's whole strip)
    // mode 3: PPL_SYM_FULL with W+- rows = a run of the packed pair index of (a <= b): plus row r <-> kplus index kp0 + r
    // (kp1: end of the run; rows up to the next multiple of 16 and the holes of the packed layout are written as zeros),
    // the minus row of the same pair is kminus(a,b) - km0; rows [rows - nzm, rows) of the launch zero the minus rows
    // zrows_m[.] (holes and the tail up to a multiple of 16), which no pair writes.
    int kp0 = 0, kp1 = 0, km0 = 0, nzm = 0;
    int zrows_m[24] = {};
    int cb_min;          // first FT-block of c that is processed (mode 2: A0 / FT; else 0)
    double *dp, *dm;     // packed outputs, row strides ldp / ldm
    int64_t ldp, ldm;
};

constexpr int FT = 32;  // (c,d) block edge of the fold

// Row bookkeeping of k_symfold: where row r of the launch reads from and which packed rows it writes.
struct FoldRow {
    int64_t roff, rowp, rowm;
    bool zero;  // write zeros (PPL_SYM_FULL rows with a > b or beyond the ragged edge)
    bool skip;  // nothing to do (amplitude rows with i > j)
};

__device__ __forceinline__ FoldRow fold_row(const FoldArgs &p, int r) {
    FoldRow f;
    f.zero = f.skip = false;
    if (p.mode == 0) {
        f.roff = (int64_t)r * p.s_row;
        f.rowp = f.rowm = r;
    } else if (p.mode == 2) {
        const int al = r / p.tbp, bl = r - al * p.tbp;
        const int a = p.A0 + al, b = p.bg0 + bl;
        f.zero = al >= p.ta || b >= p.v || a > b;
        f.roff = f.zero ? 0 : ((int64_t)al * p.rows_per_a + b - p.b_base) * p.s_row;
        f.rowp = f.rowm = r;
    } else if (p.mode == 3) {
        const int nplus = p.rows - p.nzm;
        f.zero = true;
        f.roff = 0;
        f.rowp = f.rowm = -1;
        if (r >= nplus) {  // a minus row no pair owns
            f.rowm = p.zrows_m[r - nplus];
        } else {
            f.rowp = r;
            const int64_t kap = (int64_t)p.kp0 + r;
            if (kap < p.kp1) {
                int a = p.A0 + p.ta - 1;
                while (a > p.A0 && kplus(a, a, p.v) > kap) --a;
                const int b = a + (int)(kap - kplus(a, a, p.v));
                if (b < p.v) {  // b == v: the hole in front of the next triangle row
                    f.zero = false;
                    f.roff = ((int64_t)(a - p.A0) * p.rows_per_a + b - p.b_base) * p.s_row;
                    f.rowm = a < b ? kminus(a, b, p.v) - p.km0 : -1;
                }
            }
        }
    } else {
        const int i = r / p.o, j = r - i * p.o;
        f.skip = i > j;
        f.roff = i * p.s_i + j * p.s_j - p.roff_bias;
        f.rowp = (int64_t)i * p.o - (int64_t)i * (i - 1) / 2 + (j - i);
        f.rowm = (i < j) ? (int64_t)i * (2 * p.o - i - 1) / 2 + (j - i - 1) : -1;
    }
    return f;
}

// One CTA owns one (c-block <= d-block) pair of 32 x 32 blocks and strides over the rows; the two source
// blocks of the NEXT row are fetched into registers while the current row goes through shared memory
// (transpose) and out, so that every thread keeps 8 global loads in flight across the barriers.
__global__ void __launch_bounds__(256, 4) k_symfold(const FoldArgs p) {
    __shared__ double sa[FT][FT + 1], sb[FT][FT + 1];
    const int nbv = (p.v + FT - 1) / FT;
    // blockIdx.x -> block pair (cb <= db) among the blocks cb_min..nbv-1; blockIdx.y strides over rows
    int cb = p.cb_min, rem = blockIdx.x;
    while (rem >= nbv - cb) {
        rem -= nbv - cb;
        ++cb;
    }
    const int db = cb + rem;
    const int c0 = cb * FT, d0 = db * FT;
    const int cmin = (p.mode == 2 || p.mode == 3) ? p.A0 : 0;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    const bool offdiag = cb != db;
    double va[FT / 8], vb[FT / 8];
    auto fetch = [&](const FoldRow &f) {
        const double *s = p.src + f.roff;
        const bool live = !f.zero && !f.skip;
#pragma unroll
        for (int k = 0; k < FT / 8; ++k) {
            const int y = ty + 8 * k;
            const int c = c0 + y, d = d0 + tx;
            va[k] = (live && c < p.vs && d < p.vs && c >= cmin) ? __ldg(s + (int64_t)c * p.sc + d) : 0.0;
            const int c2 = d0 + y, d2 = c0 + tx;  // the transposed block: element (c2,d2), c2 in db, d2 in cb
            vb[k] = (live && offdiag && c2 < p.vs && d2 < p.vs && d2 >= cmin) ? __ldg(s + (int64_t)c2 * p.sc + d2) : 0.0;
        }
    };
    int r = p.row0 + blockIdx.y;
    if (r >= p.rows) return;
    FoldRow cur = fold_row(p, r);
    fetch(cur);
    for (; r < p.rows; r += gridDim.y) {
        __syncthreads();  // previous row's reads of sa/sb are done
#pragma unroll
        for (int k = 0; k < FT / 8; ++k) {
            sa[ty + 8 * k][tx] = va[k];
            if (offdiag) sb[ty + 8 * k][tx] = vb[k];
        }
        const FoldRow now = cur;
        const int rn = r + gridDim.y;
        if (rn < p.rows) {
            cur = fold_row(p, rn);
            fetch(cur);
        }
        __syncthreads();
        if (now.skip) continue;
        double *op = now.rowp >= 0 ? p.dp + now.rowp * p.ldp : nullptr;
        double *om = now.rowm >= 0 ? p.dm + now.rowm * p.ldm : nullptr;
#pragma unroll
        for (int k = 0; k < FT / 8; ++k) {
            const int y = ty + 8 * k;
            const int c = c0 + y, d = d0 + tx;
            if (c >= p.v || d >= p.v || d < c || c < cmin) continue;
            const double xcd = sa[y][tx];
            if (c == d) {
                if (op) op[kplus(c, d, p.v)] = p.diag * xcd;
            } else {
                const double xdc = offdiag ? sb[tx][y] : sa[tx][y];
                if (op) op[kplus(c, d, p.v)] = p.scale * (xcd + xdc);
                if (om) om[kminus(c, d, p.v)] = p.scale * (xcd - xdc);
            }
        }
    }
}

// grid.y of a k_symfold launch: about four resident waves of CTAs (4 per SM), each CTA striding over rows
static inline int fold_grid_y(int pairs, int rows, int sms) {
    const long want = (long)sms * 4 * 4;
    long y = (want + pairs - 1) / pairs;
    if (y < 1) y = 1;
    if (y > rows) y = rows;
    if (y > 65535) y = 65535;
    return (int)y;
}

struct ReduceSaArgs {
    const double *partp, *partm;  // [sp][Mp][N], [sm][Mm][N]
    int sp, sm;
    int Mp, Mm, N;
    int o, v, tb, a0, b0;
    int mirror;                   // off-diagonal tile: also write the (b,a) entries
    double alpha, beta;
    RStrides rs;
    double *R;
};

__global__ void __launch_bounds__(256) k_reduce_sa(const ReduceSaArgs p) {
    const int64_t total = (int64_t)p.Mp * p.N;
    const int64_t MpN = total, MmN = (int64_t)p.Mm * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int mp = (int)(idx / p.N), n = (int)(idx - (int64_t)mp * p.N);
        // packed row mp -> (i <= j): i = largest with i*o - i(i-1)/2 <= mp
        int i = (int)((2.0 * p.o + 1.0 - sqrt((2.0 * p.o + 1.0) * (2.0 * p.o + 1.0) - 8.0 * mp)) * 0.5);
        while (i > 0 && (int64_t)i * p.o - (int64_t)i * (i - 1) / 2 > mp) --i;
        while ((int64_t)(i + 1) * p.o - (int64_t)(i + 1) * i / 2 <= mp) ++i;
        const int j = i + (mp - (int)((int64_t)i * p.o - (int64_t)i * (i - 1) / 2));
        double rp = 0.0, rm = 0.0;
        for (int z = 0; z < p.sp; ++z) rp += p.partp[(int64_t)z * MpN + idx];
        if (i < j) {
            const int64_t mm = (int64_t)i * (2 * p.o - i - 1) / 2 + (j - i - 1);
            const int64_t im = mm * p.N + n;
            for (int z = 0; z < p.sm; ++z) rm += p.partm[(int64_t)z * MmN + im];
        }
        const int al = n / p.tb, bl = n - al * p.tb;
        const int a = p.a0 + al, b = p.b0 + bl;
        const double v1 = rp + rm, v2 = rp - rm;  // R[i,j,a,b], R[j,i,a,b]
        r_update(p.R + i * p.rs.i + j * p.rs.j + a * p.rs.a + b * p.rs.b, v1, p.alpha, p.beta);
        if (i < j) r_update(p.R + j * p.rs.i + i * p.rs.j + a * p.rs.a + b * p.rs.b, v2, p.alpha, p.beta);
        if (p.mirror) {
            r_update(p.R + j * p.rs.i + i * p.rs.j + b * p.rs.a + a * p.rs.b, v1, p.alpha, p.beta);
            if (i < j) r_update(p.R + i * p.rs.i + j * p.rs.j + b * p.rs.a + a * p.rs.b, v2, p.alpha, p.beta);
        }
    }
}

// t2 stored 'iajb' ([i][c][j][d], the paper's 'icjd') -> [i][j][c][d] for the un-packed modes
__global__ void __launch_bounds__(256) k_permute_t2(const double *src, double *dst, int o, int v) {
    const int64_t total = (int64_t)o * o * v * v;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int d = (int)(idx % v);
        int64_t r = idx / v;
        const int c = (int)(r % v);
        r /= v;
        const int j = (int)(r % o), i = (int)(r / o);
        dst[idx] = src[(((int64_t)i * v + c) * o + j) * v + d];
    }
}

// ---------------------------------------------------------------------------------------------
// Input symmetry check (the preconditions of the symmetric modes; PAPER.md:66 for L).
// flags bit 0: L[P,a,c] != L[P,c,a]; bit 1: t2[i,j,c,d] != t2[j,i,d,c].
// Work items: for L one (P; 32 x 32 block pair ab <= cb), for t2 one (i <= j; block pair (cb, db)).  Each item loads a
// block and its partner, both along their contiguous index, and compares them through a shared-memory transpose, so
// every global read is coalesced: the check moves |L| + |t2| bytes once at HBM speed (large: 4 GB, ~0.7 ms).
// ---------------------------------------------------------------------------------------------
struct CheckArgs {
    const double *L, *t2;  // either may be null (not checked)
    int o, v, x;
    int64_t s_i, s_j, s_c;  // element strides of t2[i][j][c][.] (d contiguous) in the caller's storage order
    volatile int *flags;    // [2] in MAPPED PINNED HOST memory, cleared by the host before the launch: [0] = 1 if L is not symmetric,
                            // [1] = 1 if t2 is not pair-symmetric.  Plain stores of the same value (no atomics across PCIe, no
                            // device-to-host copy behind the kernel): the host reads them once the kernel's event has completed.
};
// The scan of block `bid` of `nblocks` (any block size that is a multiple of 32; sb: 32 x 33 doubles of shared memory); returns the
// flag bits this thread found.  Shared by k_check_inputs and by the one-kernel path of launch-bound shapes, whose first few
// CTAs run it (ppl_kernels_small.cuh).
__device__ __forceinline__ int check_inputs_scan(const CheckArgs &p, double (*sb)[33], int bid, int nblocks) {
    const int nb = (p.v + 31) / 32;
    const int64_t npair = (int64_t)nb * (nb + 1) / 2, nsq = (int64_t)nb * nb;
    const int64_t itemsL = p.L ? (int64_t)p.x * npair : 0;
    const int64_t itemsT = p.t2 ? (int64_t)p.o * (p.o + 1) / 2 * nsq : 0;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, nty = blockDim.x >> 5;
    int f = 0;
    for (int64_t item = bid; item < itemsL + itemsT; item += nblocks) {
        const double *A, *B;  // block of A at (r0, c0) is compared with the transpose of the block of B at (c0, r0)
        int64_t lda, ldb;
        int r0, c0, bit;
        bool diag;
        if (item < itemsL) {
            const int64_t P = item / npair;
            int rem = (int)(item - P * npair), rb = 0;
            while (rem >= nb - rb) {
                rem -= nb - rb;
                ++rb;
            }
            A = B = p.L + P * (int64_t)p.v * p.v;
            lda = ldb = p.v;
            r0 = rb * 32;
            c0 = (rb + rem) * 32;
            bit = 1;
            diag = rem == 0;
        } else {
            const int64_t e = item - itemsL, ij = e / nsq;
            const int blk = (int)(e - ij * nsq);
            int i = 0;
            int64_t rem = ij;
            while (rem >= p.o - i) {
                rem -= p.o - i;
                ++i;
            }
            const int j = i + (int)rem;
            A = p.t2 + i * p.s_i + j * p.s_j;
            B = p.t2 + j * p.s_i + i * p.s_j;
            lda = ldb = p.s_c;
            r0 = (blk / nb) * 32;
            c0 = (blk % nb) * 32;
            bit = 2;
            diag = false;
        }
        __syncthreads();  // the previous item's reads of sb are done
        for (int y = ty; y < 32; y += nty) {
            const int r = c0 + y, c = r0 + tx;  // partner block: rows c0.., columns r0..
            sb[y][tx] = (r < p.v && c < p.v) ? __ldg(B + (int64_t)r * ldb + c) : 0.0;
        }
        __syncthreads();
        for (int y = ty; y < 32; y += nty) {
            const int r = r0 + y, c = c0 + tx;
            if (r < p.v && c < p.v && !(diag && c < r)) {
                if (__ldg(A + (int64_t)r * lda + c) != sb[tx][y]) f |= bit;
            }
        }
    }
    return f;
}
__global__ void __launch_bounds__(256) k_check_inputs(const CheckArgs p) {
    __shared__ double sb[32][33];
    const int f = check_inputs_scan(p, sb, blockIdx.x, gridDim.x);
    if (f & 1) p.flags[0] = 1;
    if (f & 2) p.flags[1] = 1;
}

// ppl_apply_host in PPL_SYM_FULL: t2 never sits on the device whole, so k_check_inputs cannot compare row (i,j) with row
// (j,i).  The packing uses the rows i <= j only; this kernel looks at the OTHER rows of a staged chunk, which the path
// would otherwise never read:
//   i == j:  t2[i,i,c,d] == t2[i,i,d,c] directly (the antisymmetric part of a diagonal row has no place in tau-);
//   i >  j:  the row folded as its mirror image must reproduce, bit for bit, what row (j,i) wrote into tau+- earlier
//            (chunks arrive in ascending (i,j), and (j,i) < (i,j)):
//                tau+[(j,i)][(c,d)] == scale (x[c,d] + x[d,c]),   tau-[(j,i)][(c,d)] == scale (x[d,c] - x[c,d]),   x = t2[i,j,.,.]
//            -- the same two operands in the same operations as k_symfold, so a pair-symmetric t2 passes exactly, and a
//            t2 that passes differs from a pair-symmetric one by at most the rounding of those sums.
// One item = one such row x one pair (c-block <= d-block) of 32 x 32 blocks, staged through shared memory as in
// check_inputs_scan so that both the block and its transpose are read coalesced.
struct CheckRowsArgs {
    const double *t2;       // the staged chunk: rows [row0, row1) of the dense [i][j][c][d] array, row row0 first
    const double *taup, *taum;
    int64_t ldp, ldm;
    int row0, row1;         // rows of the flattened (i,j) index held by the staged chunk
    int o, v, vp;           // v: nvirt of the source; vp: nvirt of the packed geometry (kplus / kminus)
    double scale, diag;     // the factors the chunk was packed with (k_symfold)
    volatile int *flags;    // as CheckArgs::flags; only [1] is written here
};
__global__ void __launch_bounds__(256) k_check_t2_rows(const CheckRowsArgs p) {
    __shared__ double sa[32][33], sb[32][33];
    const int nb = (p.v + 31) / 32;
    const int64_t npair = (int64_t)nb * (nb + 1) / 2;
    const int64_t items = (int64_t)(p.row1 - p.row0) * npair;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t vv = (int64_t)p.v * p.v;
    bool bad = false;
    for (int64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const int r = p.row0 + (int)(item / npair);
        const int i = r / p.o, j = r - i * p.o;
        if (i < j) continue;  // (uniform over the block) rows the packing itself reads
        int rem = (int)(item % npair), cb = 0;
        while (rem >= nb - cb) {
            rem -= nb - cb;
            ++cb;
        }
        const int c0 = cb * 32, d0 = (cb + rem) * 32;
        const double *x = p.t2 + (int64_t)(r - p.row0) * vv;
        __syncthreads();  // the previous item's reads of sa / sb are done
        for (int y = ty; y < 32; y += 8) {
            const int c = c0 + y, d = d0 + tx;
            sa[y][tx] = (c < p.v && d < p.v) ? __ldg(x + (int64_t)c * p.v + d) : 0.0;
            const int c2 = d0 + y, d2 = c0 + tx;
            sb[y][tx] = (c2 < p.v && d2 < p.v) ? __ldg(x + (int64_t)c2 * p.v + d2) : 0.0;
        }
        __syncthreads();
        const double *tp = p.taup + rowplus(j, i, p.o) * p.ldp;
        const double *tm = i > j ? p.taum + rowminus(j, i, p.o) * p.ldm : nullptr;
        for (int y = ty; y < 32; y += 8) {
            const int c = c0 + y, d = d0 + tx;
            if (c >= p.v || d >= p.v || d < c) continue;
            const double xcd = sa[y][tx], xdc = sb[tx][y];
            if (i == j) {
                if (xcd != xdc) bad = true;
            } else if (c == d) {
                if (tp[kplus(c, d, p.vp)] != p.diag * xcd) bad = true;
            } else {
                if (tp[kplus(c, d, p.vp)] != p.scale * (xcd + xdc)) bad = true;
                if (tm[kminus(c, d, p.vp)] != p.scale * (xdc - xcd)) bad = true;
            }
        }
    }
    if (bad) p.flags[1] = 1;
}

// ---------------------------------------------------------------------------------------------
// FP64 tensor-pipe peak probe (register-only DMMA stream) and a one-warp fragment-layout check
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512, 1) k_probe_dmma(double *out, int iters, double a, double b) {
    double d0[8], d1[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        d0[i] = threadIdx.x * 1e-3 + i;
        d1[i] = i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma(d0[i], d1[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += d0[i] + d1[i];
    if (s == 123.456) out[0] = s;  // never true; keeps the loop alive
}

// Variants of the probe that back the pipe choice (north_star: "DMMA or the FP64 FMA pipe, whichever is faster";
// DESIGN.md section 6, profiles/r02_fp64_peaks.md).  ACC independent accumulator chains per warp (DMMA) or per
// thread (DFMA); MIX interleaves one DFMA chain step per DMMA.  flops per iteration and warp:
//   DMMA: ACC * 512;  DFMA: ACC * 2 * 32;  MIX: ACC * (512 + 64).
template <int ACC>
__global__ void __launch_bounds__(512, 1) k_probe_dmma_n(double *out, int iters, double a, double b) {
    double d0[ACC], d1[ACC];
#pragma unroll
    for (int i = 0; i < ACC; ++i) {
        d0[i] = threadIdx.x * 1e-3 + i;
        d1[i] = i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ACC; ++i) dmma(d0[i], d1[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ACC; ++i) s += d0[i] + d1[i];
    if (s == 123.456) out[0] = s;
}

template <int ACC>
__global__ void __launch_bounds__(512, 1) k_probe_dfma(double *out, int iters, double a, double b) {
    double f[ACC];
#pragma unroll
    for (int i = 0; i < ACC; ++i) f[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ACC; ++i) f[i] = fma(f[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ACC; ++i) s += f[i];
    if (s == 123.456) out[0] = s;
}

template <int ACC>
__global__ void __launch_bounds__(512, 1) k_probe_mix(double *out, int iters, double a, double b) {
    double d0[ACC], d1[ACC], f[ACC];
#pragma unroll
    for (int i = 0; i < ACC; ++i) {
        d0[i] = threadIdx.x * 1e-3 + i;
        d1[i] = i;
        f[i] = 0.5 * i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ACC; ++i) {
            dmma(d0[i], d1[i], a, b);
            f[i] = fma(f[i], a, b);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ACC; ++i) s += d0[i] + d1[i] + f[i];
    if (s == 123.456) out[0] = s;
}

// C(8x8) = A(8x4, row-major) * B(4x8, row-major) with one warp, using the layout stated above
__global__ void k_dmma_layout(const double *A, const double *B, double *C) {
    const int lane = threadIdx.x, g = lane >> 2, q = lane & 3;
    double c0 = 0.0, c1 = 0.0;
    dmma(c0, c1, A[g * 4 + q], B[q * 8 + g]);
    C[g * 8 + 2 * q] = c0;
    C[g * 8 + 2 * q + 1] = c1;
}

}  // namespace ppl
