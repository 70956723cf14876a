// ppl_contract.cu -- the generic pair contraction 'op0,op1->out' of the paper's generic recipe:
//
//     C[out] = beta * C[out] + alpha * sum_{summed letters} A[op0] * B[op1]            (FP64, dense row-major operands)
//
// for any two-operand contraction of tensordot type (every letter occurs in exactly two of op0, op1, out; the paper's
// "a...,b...->a..b.."), e.g. the ladder's own steps 'xac,xbd->acbd' and 'abcd,ecfd->efab'.
//
// The paper moves such a contraction through VRAM in host-driven batches along the surviving (non-summed) axes and calls
// tensordot -- i.e. permuted copies plus a library DGEMM -- per batch (Table 1 mem(generic)).  Here the
// operands are resident and nothing is permuted or copied: the contraction is ONE GEMM  C[m][n] = sum_k A[m][k] B[n][k]
// whose rows m run over the surviving letters of op0, columns n over those of op1 and k over the summed letters, with
// every operand addressed in place through offset tables ("block-scatter" addressing: element (m, k) of A sits at
// offAm[m] + offAk[k]).  The batches of the paper are the CTA tiles (128 m x 128 n): always along surviving axes; the
// summed axes (the Cholesky index x among them) are never split across launches -- only inside the kernel (split-K with
// a fixed-order reduction, so results are bit-reproducible).  Tiles are staged global -> shared with cp.async (16-byte
// where an operand's unit-stride letter allows, else 8-byte), a 4-stage ring, and multiplied on the FP64 tensor pipe
// (DMMA m8n8k4) with the accumulators in registers.
#include "../../include/ppl.h"
#include "ppl_device.cuh"
#include "ppl_internal.h"

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <vector>

namespace ppl {

constexpr int GLD_MN = BM + 4;  // row stride of a [k][m] tile (doubles): 16-byte aligned rows, conflict-free LDS.64
constexpr int GLD_K = BK + 4;   // row stride of a [m][k] tile
constexpr int GTILE = (BK * GLD_MN > BM * GLD_K) ? BK * GLD_MN : BM * GLD_K;  // doubles per operand tile per stage
constexpr size_t SMEM_GATHER = (size_t)STAGES * 2 * GTILE * sizeof(double);

struct ContractArgs {
    const double *A, *B;
    double *C;
    const int64_t *offAm, *offAk, *offBn, *offBk, *offCm, *offCn;  // element offsets
    int M, N, K;
    int a_vec, b_vec;   // 1: pairs along the operand's unit-stride direction may be fetched with one 16-byte copy
    int k_per_split;    // multiple of BK
    int splitk;
    double *part;       // splitk > 1: [splitk][M][N]
    double alpha, beta;
};

// One operand tile: 128 rows (m or n) x 16 k.  KFAST: the operand's unit-stride letter is a summed one -> smem [row][k]
// (stride GLD_K), threads run along k; else smem [k][row] (stride GLD_MN), threads run along the rows.
template <bool KFAST>
__device__ __forceinline__ void gather_tile(double *s, const double *g, const int64_t *offR, const int64_t *offK, int r0, int R,
                                            int k0, int Kend, bool vec, int tid) {
    if (KFAST) {
        if (vec) {  // 8 pairs per row
#pragma unroll
            for (int c = 0; c < (BM * BK / 2) / NTHREADS; ++c) {
                const int idx = tid + c * NTHREADS, row = idx >> 3, k = (idx & 7) << 1;
                const bool ok = r0 + row < R && k0 + k < Kend;  // Kend and k0 + k even: the pair is in or out as one
                const double *src = ok ? g + offR[r0 + row] + offK[k0 + k] : g;
                cp_async16(s + row * GLD_K + k, src, ok ? 16 : 0);
            }
        } else {
#pragma unroll
            for (int c = 0; c < (BM * BK) / NTHREADS; ++c) {
                const int idx = tid + c * NTHREADS, row = idx >> 4, k = idx & 15;
                const bool ok = r0 + row < R && k0 + k < Kend;
                const double *src = ok ? g + offR[r0 + row] + offK[k0 + k] : g;
                cp_async8(s + row * GLD_K + k, src, ok ? 8 : 0);
            }
        }
    } else {
        if (vec) {  // 64 pairs per k
#pragma unroll
            for (int c = 0; c < (BM * BK / 2) / NTHREADS; ++c) {
                const int idx = tid + c * NTHREADS, k = idx >> 6, row = (idx & 63) << 1;
                const bool ok = r0 + row < R && k0 + k < Kend;  // R even when vec
                const double *src = ok ? g + offR[r0 + row] + offK[k0 + k] : g;
                cp_async16(s + k * GLD_MN + row, src, ok ? 16 : 0);
            }
        } else {
#pragma unroll
            for (int c = 0; c < (BM * BK) / NTHREADS; ++c) {
                const int idx = tid + c * NTHREADS, k = idx >> 7, row = idx & 127;
                const bool ok = r0 + row < R && k0 + k < Kend;
                const double *src = ok ? g + offR[r0 + row] + offK[k0 + k] : g;
                cp_async8(s + k * GLD_MN + row, src, ok ? 8 : 0);
            }
        }
    }
}

template <bool AKF, bool BKF>
__global__ void __launch_bounds__(NTHREADS, 1) k_contract_gather(const ContractArgs p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *As = reinterpret_cast<double *>(smem_raw);
    double *Bs = As + STAGES * GTILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    const int tiles_m = (p.M + BM - 1) / BM, tiles_n = (p.N + BN - 1) / BN;
    int tm, tn;
    raster(blockIdx.x, tiles_m, tiles_n, tm, tn);
    const int m0 = tm * BM, n0 = tn * BN;
    const int z = blockIdx.y;
    const int Kbeg = z * p.k_per_split, Kend = min(p.K, Kbeg + p.k_per_split);
    const int nkt = max(0, (Kend - Kbeg + BK - 1) / BK);

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) {
            gather_tile<AKF>(As + s * GTILE, p.A, p.offAm, p.offAk, m0, p.M, Kbeg + s * BK, Kend, p.a_vec != 0, tid);
            gather_tile<BKF>(Bs + s * GTILE, p.B, p.offBn, p.offBk, n0, p.N, Kbeg + s * BK, Kend, p.b_vec != 0, tid);
        }
        cp_async_commit();
    }
    // element (row, kk) of a stage tile
    constexpr int a_sr = AKF ? GLD_K : 1, a_sk = AKF ? 1 : GLD_MN;
    constexpr int b_sr = BKF ? GLD_K : 1, b_sk = BKF ? 1 : GLD_MN;
    for (int kt = 0; kt < nkt; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int kn = kt + STAGES - 1;
            if (kn < nkt) {
                const int s = kn % STAGES;
                gather_tile<AKF>(As + s * GTILE, p.A, p.offAm, p.offAk, m0, p.M, Kbeg + kn * BK, Kend, p.a_vec != 0, tid);
                gather_tile<BKF>(Bs + s * GTILE, p.B, p.offBn, p.offBk, n0, p.N, Kbeg + kn * BK, Kend, p.b_vec != 0, tid);
            }
            cp_async_commit();
        }
        const double *as = As + (kt % STAGES) * GTILE + (wm * WTM + g) * a_sr;
        const double *bs = Bs + (kt % STAGES) * GTILE + (wn * WTN + g) * b_sr;
#pragma unroll
        for (int k4 = 0; k4 < BK / 4; ++k4) {
            const int kk = k4 * 4 + q;
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = as[i * 8 * a_sr + kk * a_sk];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = bs[j * 8 * b_sr + kk * b_sk];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

    // epilogue: block (i,j): row g <-> m = mw + 8i + g; cols n = nw + 8j + 2q, +1
    if (p.splitk > 1) {
        double *part = p.part + (int64_t)z * p.M * p.N;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int m = m0 + wm * WTM + 8 * i + g;
            if (m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int n = n0 + wn * WTN + 8 * j + 2 * q;
                if (n < p.N) part[(int64_t)m * p.N + n] = acc[i][j][0];
                if (n + 1 < p.N) part[(int64_t)m * p.N + n + 1] = acc[i][j][1];
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int m = m0 + wm * WTM + 8 * i + g;
            if (m >= p.M) continue;
            double *crow = p.C + p.offCm[m];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int n = n0 + wn * WTN + 8 * j + 2 * q;
                if (n < p.N) r_update(crow + p.offCn[n], acc[i][j][0], p.alpha, p.beta);
                if (n + 1 < p.N) r_update(crow + p.offCn[n + 1], acc[i][j][1], p.alpha, p.beta);
            }
        }
    }
}

// fixed-order sum of the split-K partials, then C = beta C + alpha sum
__global__ void __launch_bounds__(256) k_contract_reduce(const ContractArgs p) {
    const int64_t MN = (int64_t)p.M * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < MN; idx += (int64_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int zz = 0; zz < p.splitk; ++zz) s += p.part[(int64_t)zz * MN + idx];
        const int m = (int)(idx / p.N), n = (int)(idx - (int64_t)m * p.N);
        r_update(p.C + p.offCm[m] + p.offCn[n], s, p.alpha, p.beta);
    }
}

// The six offset tables of a request are computed ON THE DEVICE from the <= 12 extents and strides of each axis group
// (kernel parameters: no host table, no upload, nothing that blocks the host or a stream capture).
struct AxisGroup {       // one offset table: the flattened index over n letters, last letter fastest
    int64_t ext[12], stride[12];
    int64_t count;         // product of the extents (1 when n == 0)
    int32_t n, pad_;
};
struct AxisTables {
    AxisGroup t[6];      // in workspace order: A rows, C rows, B columns, C columns, A k, B k
};

__global__ void __launch_bounds__(256) k_fill_tables(const AxisTables f, int64_t *tab) {
    int64_t total = 0;
    for (int w = 0; w < 6; ++w) total += f.t[w].count;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        int64_t r = idx;
        int w = 0;
        while (r >= f.t[w].count) r -= f.t[w++].count;
        const AxisGroup &ax = f.t[w];
        int64_t off = 0;
        for (int k = ax.n - 1; k >= 0; --k) {
            const int64_t q = r / ax.ext[k];
            off += (r - q * ax.ext[k]) * ax.stride[k];
            r = q;
        }
        tab[idx] = off;
    }
}

}  // namespace ppl

namespace {

struct Parsed {
    std::vector<char> op[3];
    int64_t ext[128];
    std::vector<char> Ml, Nl, Kl;  // surviving letters of op0 / op1 (in their operand's order), summed letters (in op0's order)
    int64_t M = 1, N = 1, K = 1;
};

// "op0,op1->out": letters only, none repeated inside one operand, every letter in exactly two of the three
int parse(const char *subs, const int64_t *dims0, const int64_t *dims1, Parsed *ps) {
    if (!subs || !dims0 || !dims1) return PPL_ERR_INVALID_ARG;
    int which = 0;
    for (const char *q = subs; *q; ++q) {
        const char ch = *q;
        if (ch == ' ') continue;
        if (ch == ',') {
            if (which != 0) return PPL_ERR_INVALID_ARG;
            which = 1;
        } else if (ch == '-' && q[1] == '>') {
            if (which != 1) return PPL_ERR_INVALID_ARG;
            which = 2;
            ++q;
        } else if ((ch >= 'a' && ch <= 'z') || (ch >= 'A' && ch <= 'Z')) {
            for (char c : ps->op[which])
                if (c == ch) return PPL_ERR_INVALID_ARG;
            if (ps->op[which].size() >= 12) return PPL_ERR_INVALID_ARG;
            ps->op[which].push_back(ch);
        } else {
            return PPL_ERR_INVALID_ARG;
        }
    }
    if (which != 2) return PPL_ERR_INVALID_ARG;
    for (int k = 0; k < 128; ++k) ps->ext[k] = 0;
    auto has = [&](int w, char c) { return std::find(ps->op[w].begin(), ps->op[w].end(), c) != ps->op[w].end(); };
    for (size_t k = 0; k < ps->op[0].size(); ++k) {
        if (dims0[k] < 1) return PPL_ERR_INVALID_ARG;
        ps->ext[(int)ps->op[0][k]] = dims0[k];
    }
    for (size_t k = 0; k < ps->op[1].size(); ++k) {
        const char c = ps->op[1][k];
        if (dims1[k] < 1 || (has(0, c) && ps->ext[(int)c] != dims1[k])) return PPL_ERR_INVALID_ARG;
        ps->ext[(int)c] = dims1[k];
    }
    for (char c : ps->op[0]) {
        if (has(1, c) == has(2, c)) return PPL_ERR_INVALID_ARG;  // in all three (batch letter) or in op0 alone
        (has(1, c) ? ps->Kl : ps->Ml).push_back(c);
    }
    for (char c : ps->op[1]) {
        if (has(0, c) == has(2, c)) return PPL_ERR_INVALID_ARG;
        if (!has(0, c)) ps->Nl.push_back(c);
    }
    for (char c : ps->op[2])
        if (!has(0, c) && !has(1, c)) return PPL_ERR_INVALID_ARG;
    if (ps->op[2].size() != ps->Ml.size() + ps->Nl.size()) return PPL_ERR_INVALID_ARG;
    for (char c : ps->Ml) ps->M *= ps->ext[(int)c];
    for (char c : ps->Nl) ps->N *= ps->ext[(int)c];
    for (char c : ps->Kl) ps->K *= ps->ext[(int)c];
    const int64_t lim = INT32_MAX / 2;
    if (ps->M > lim || ps->N > lim || ps->K > lim) return PPL_ERR_INVALID_ARG;
    return PPL_OK;
}

// element stride of letter c in a dense row-major array with subscripts `op`
int64_t stride_of(const std::vector<char> &op, const int64_t *ext, char c) {
    int64_t s = 1;
    for (size_t k = op.size(); k-- > 0;) {
        if (op[k] == c) return s;
        s *= ext[(int)op[k]];
    }
    return 0;
}

// One axis group of the request: the letters of `letters` as they sit in the array with subscripts `op`
void axis_group(const std::vector<char> &letters, const std::vector<char> &op, const int64_t *ext, ppl::AxisGroup *ax) {
    ax->n = (int32_t)letters.size();
    ax->pad_ = 0;
    ax->count = 1;
    for (int k = 0; k < 12; ++k) ax->ext[k] = 1, ax->stride[k] = 0;
    for (size_t k = 0; k < letters.size(); ++k) {
        ax->ext[k] = ext[(int)letters[k]];
        ax->stride[k] = stride_of(op, ext, letters[k]);
        ax->count *= ax->ext[k];
    }
}
// the six tables in workspace order: rows of A / C over the surviving letters of op0, columns of B / C over those of op1,
// k over the summed letters (in op0's order for both operands)
enum { T_AM = 0, T_CM, T_BN, T_CN, T_AK, T_BK };
void axis_tables(const Parsed &ps, ppl::AxisTables *f) {
    axis_group(ps.Ml, ps.op[0], ps.ext, &f->t[T_AM]);
    axis_group(ps.Ml, ps.op[2], ps.ext, &f->t[T_CM]);
    axis_group(ps.Nl, ps.op[1], ps.ext, &f->t[T_BN]);
    axis_group(ps.Nl, ps.op[2], ps.ext, &f->t[T_CN]);
    axis_group(ps.Kl, ps.op[0], ps.ext, &f->t[T_AK]);
    axis_group(ps.Kl, ps.op[1], ps.ext, &f->t[T_BK]);
}

// Along `run`, are the elements (2i, 2i+1) neighbours in memory at an even element offset (a 16-byte aligned pair),
// whatever the position along `other`?  Fold the trailing letters of `run` that are contiguous with each other into
// one group; it must have stride 1 and an even extent, and every other letter with more than one value (of `run` and of
// `other`) must have an even stride.  (An odd group cannot work: the pair straddling its end would need the next
// letter's stride to equal the group's extent, i.e. the next letter would belong to the group.)
bool pairs_ok(const ppl::AxisGroup &run, const ppl::AxisGroup &other, const void *base) {
    if (((uintptr_t)base & 15) != 0 || (run.count & 1)) return false;
    int k = run.n - 1;
    while (k >= 0 && run.ext[k] == 1) --k;
    if (k < 0 || run.stride[k] != 1) return false;
    int64_t group = run.ext[k];
    for (--k; k >= 0; --k) {
        if (run.ext[k] == 1) continue;
        if (run.stride[k] != group) break;  // not contiguous with the group so far
        group *= run.ext[k];
    }
    if (group & 1) return false;
    for (; k >= 0; --k)
        if (run.ext[k] > 1 && (run.stride[k] & 1)) return false;
    for (int j = 0; j < other.n; ++j)
        if (other.ext[j] > 1 && (other.stride[j] & 1)) return false;
    return true;
}
// offset(i) == i * stride for every i of the group?  (all letters with more than one value contiguous with each other)
bool affine(const ppl::AxisGroup &g, int64_t stride) {
    int64_t want = stride;
    for (int k = g.n - 1; k >= 0; --k) {
        if (g.ext[k] == 1) continue;
        if (g.stride[k] != want) return false;
        want *= g.ext[k];
    }
    return true;
}
// Plain matrix pairs that go to the persistent TMA kernels of the ladder (34-35 TFLOP/s):
//   K_OUTER  A[K][M], B[K][N], C[M][N] all dense in that order (the paper's step 0 'xac,xbd->acbd'): k_step0_tma
//   K_INNER  A[M][K], B[N][K] dense (its step 1 with t2 stored [e,f,c,d], 'abcd,efcd->efab'): k_step1_tma into split-K
//            partials, then the table-driven reduction scatters into C in any order
enum Route { GENERIC = 0, K_OUTER, K_INNER };
Route classify(const Parsed &ps, const ppl::AxisTables &f) {
    if (!(ps.M & 1) && !(ps.N & 1) && affine(f.t[T_AK], ps.M) && affine(f.t[T_AM], 1) && affine(f.t[T_BK], ps.N) &&
        affine(f.t[T_BN], 1) && affine(f.t[T_CM], ps.N) && affine(f.t[T_CN], 1))
        return K_OUTER;
    if (!(ps.K & 1) && affine(f.t[T_AM], ps.K) && affine(f.t[T_AK], 1) && affine(f.t[T_BN], ps.K) && affine(f.t[T_BK], 1)) return K_INNER;
    return GENERIC;
}

size_t table_bytes(const Parsed &ps) { return (size_t)(2 * ps.M + 2 * ps.N + 2 * ps.K) * sizeof(int64_t); }

// split-K factor: the estimated time of the launch -- whole waves of CTA tiles on `sms` SMs, each (k-tiles + pipeline
// fill) long, plus writing and re-reading the partials -- minimised over the factors whose partials fit into `room`
int pick_splitk(const Parsed &ps, int sms, size_t room) {
    const int64_t tiles = ((ps.M + ppl::BM - 1) / ppl::BM) * ((ps.N + ppl::BN - 1) / ppl::BN);
    const int64_t nkt = (ps.K + ppl::BK - 1) / ppl::BK;
    const double tau = 2.0 * ppl::BM * ppl::BN * ppl::BK / (37.2e12 / sms);  // one k-tile on one SM
    int best = 1;
    double best_t = 1e300;
    const int64_t smax = std::max<int64_t>(1, std::min<int64_t>(nkt / 8, 64));
    for (int64_t s = 1; s <= smax; ++s) {
        const int64_t kt_per = (nkt + s - 1) / s;
        if ((nkt + kt_per - 1) / kt_per != s) continue;  // no empty splits
        if (s > 1 && (size_t)s * ps.M * ps.N * 8 > room) break;
        const double waves = (double)((tiles * s + sms - 1) / sms);
        const double t = waves * (kt_per + 6) * tau + (s > 1 ? (double)(s + 2) * ps.M * ps.N * 8.0 / 6.0e12 + 4e-6 : 0.0);
        if (t < best_t) {
            best_t = t;
            best = (int)s;
        }
    }
    return best;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// ppl_contract_pair_noalloc: the same contraction for callers that must not allocate device memory (include/ppl.h).
//
// Everything the gather GEMM needs beyond A, B and C -- the six offset tables and, when the summed range is split, the
// split-K partials -- lives in ONE fixed array that is part of the library image.  The driver places it on every
// device that loads this library's code and keeps it there until the process exits; PPL_NOALLOC_SCRATCH_BYTES is the
// whole price, paid once, and also the hard limit of what a request may need.
//
// In host code the identifier `noalloc_scratch` is only the host-side handle of that array, not something a kernel
// may dereference: the device address comes from cudaGetSymbolAddress, asked for once per device (with that device
// current) in contract_device() below, and it is that address which the kernels receive.
//
// The tables are written by a small kernel from the <= 12 extents and strides of each axis group (kernel parameters:
// no host table, no upload), so a call is three launches at most and touches no allocator, on the host side of CUDA or
// on the device.  Every call rewrites every word of the array it later reads (all tables; all M x N entries of every
// partial), so nothing has to be cleared between calls; what the previous call left there is simply overwritten.
// All calls on a device share the array: two calls whose kernels can overlap on the GPU (different streams with no
// dependency between them, or two host threads) race on it.  Calls on one stream are ordered and safe.
namespace ppl {

static __device__ __align__(256) unsigned char noalloc_scratch[PPL_NOALLOC_SCRATCH_BYTES];

}  // namespace ppl

namespace {

// Per-device facts every call needs, looked up once (with that device current) and cached: compute capability, SM count,
// the gather kernels' shared-memory opt-in, and -- for ppl_contract_pair_noalloc only -- the device address of the
// library's built-in scratch array.  No cudaGetDeviceProperties (a slow driver query) on any per-call path.
struct ContractDevice {
    bool ready = false;
    int sms = 0;
    unsigned char *scratch = nullptr;  // DEVICE address of ppl::noalloc_scratch on this device (set by the no-alloc entry point)
};
std::mutex contract_mutex;
ContractDevice contract_dev[64];

int contract_device(const ContractDevice **out, bool want_scratch) {
    int dev = -1, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64 ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
        (void)cudaGetLastError();
        return PPL_ERR_UNSUPPORTED_DEVICE;
    }
    std::lock_guard<std::mutex> lock(contract_mutex);
    ContractDevice &d = contract_dev[dev];
    if (!d.ready) {
        bool ok = cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && d.sms > 0;
        ok = ok && cudaFuncSetAttribute(ppl::k_contract_gather<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_GATHER) == cudaSuccess;
        ok = ok && cudaFuncSetAttribute(ppl::k_contract_gather<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_GATHER) == cudaSuccess;
        ok = ok && cudaFuncSetAttribute(ppl::k_contract_gather<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_GATHER) == cudaSuccess;
        ok = ok && cudaFuncSetAttribute(ppl::k_contract_gather<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_GATHER) == cudaSuccess;
        if (!ok) {
            (void)cudaGetLastError();
            return PPL_ERR_CUDA;
        }
        d.ready = true;
    }
    if (want_scratch && !d.scratch) {
        // In host code `ppl::noalloc_scratch` is only the host-side handle of the array; a kernel needs its device address.
        unsigned char *ptr = nullptr;
        if (cudaGetSymbolAddress((void **)&ptr, ppl::noalloc_scratch) != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            return PPL_ERR_CUDA;
        }
        d.scratch = ptr;
    }
    *out = &d;
    return PPL_OK;
}

// tables -> `tab` on the device, and the launch of the gather GEMM (+ the fixed-order reduction when it splits k) with
// its partials at `part` (room bytes)
int launch_fill(const Parsed &ps, const ppl::AxisTables &f, int64_t *tab, int sms, cudaStream_t stream) {
    const int64_t entries = 2 * (ps.M + ps.N + ps.K);
    ppl::k_fill_tables<<<(int)std::min<int64_t>((entries + 255) / 256, (int64_t)sms * 8), 256, 0, stream>>>(f, tab);
    return cudaGetLastError() == cudaSuccess ? PPL_OK : PPL_ERR_CUDA;
}
void table_pointers(const Parsed &ps, const int64_t *tab, ppl::ContractArgs *a) {
    a->offAm = tab;
    a->offCm = a->offAm + ps.M;
    a->offBn = a->offCm + ps.M;
    a->offCn = a->offBn + ps.N;
    a->offAk = a->offCn + ps.N;
    a->offBk = a->offAk + ps.K;
    a->M = (int)ps.M;
    a->N = (int)ps.N;
    a->K = (int)ps.K;
}
bool kfast(const Parsed &ps, int which) {  // does operand `which` run in memory along a summed letter?
    return !ps.op[which].empty() && std::find(ps.Kl.begin(), ps.Kl.end(), ps.op[which].back()) != ps.Kl.end();
}
int launch_gather(const Parsed &ps, const ppl::AxisTables &f, ppl::ContractArgs a, unsigned char *part, size_t room, int sms,
                  cudaStream_t stream) {
    const bool a_kfast = kfast(ps, 0), b_kfast = kfast(ps, 1);
    a.a_vec = a_kfast ? pairs_ok(f.t[T_AK], f.t[T_AM], a.A) : pairs_ok(f.t[T_AM], f.t[T_AK], a.A);
    a.b_vec = b_kfast ? pairs_ok(f.t[T_BK], f.t[T_BN], a.B) : pairs_ok(f.t[T_BN], f.t[T_BK], a.B);
    a.splitk = pick_splitk(ps, sms, room);
    const int64_t nkt = (ps.K + ppl::BK - 1) / ppl::BK;
    const int64_t kt_per = (nkt + a.splitk - 1) / a.splitk;
    a.splitk = (int)((nkt + kt_per - 1) / kt_per);  // no empty splits
    a.k_per_split = (int)(kt_per * ppl::BK);
    a.part = a.splitk > 1 ? reinterpret_cast<double *>(part) : nullptr;
    const int64_t tiles = ((ps.M + ppl::BM - 1) / ppl::BM) * ((ps.N + ppl::BN - 1) / ppl::BN);
    if (tiles > INT32_MAX) return PPL_ERR_INVALID_ARG;
    const dim3 grid((unsigned)tiles, (unsigned)a.splitk);
    if (a_kfast && b_kfast)
        ppl::k_contract_gather<true, true><<<grid, ppl::NTHREADS, ppl::SMEM_GATHER, stream>>>(a);
    else if (a_kfast)
        ppl::k_contract_gather<true, false><<<grid, ppl::NTHREADS, ppl::SMEM_GATHER, stream>>>(a);
    else if (b_kfast)
        ppl::k_contract_gather<false, true><<<grid, ppl::NTHREADS, ppl::SMEM_GATHER, stream>>>(a);
    else
        ppl::k_contract_gather<false, false><<<grid, ppl::NTHREADS, ppl::SMEM_GATHER, stream>>>(a);
    if (cudaGetLastError() != cudaSuccess) return PPL_ERR_CUDA;
    if (a.splitk > 1) {
        const int64_t MN = ps.M * ps.N;
        ppl::k_contract_reduce<<<(int)std::min<int64_t>((MN + 255) / 256, (int64_t)sms * 8), 256, 0, stream>>>(a);
        if (cudaGetLastError() != cudaSuccess) return PPL_ERR_CUDA;
    }
    return PPL_OK;
}

}  // namespace

extern "C" {

int ppl_contract_pair_workspace(const char *subscripts, const int64_t *dims0, const int64_t *dims1, size_t *bytes) {
    Parsed ps;
    const int rc = parse(subscripts, dims0, dims1, &ps);
    if (rc != PPL_OK || !bytes) return ppl_fail_code(rc != PPL_OK ? rc : PPL_ERR_INVALID_ARG);
    ppl::AxisTables f;
    axis_tables(ps, &f);
    const Route route = classify(ps, f);
    // the SM count of the current device when there is one (the split-K estimate depends on it), else a B200's 148
    const ContractDevice *dev = nullptr;
    const int sms = contract_device(&dev, false) == PPL_OK ? dev->sms : 148;
    const int s = pick_splitk(ps, sms, ~(size_t)0);
    size_t part = 0;  // K_OUTER writes C directly; K_INNER always goes through partials; GENERIC only when it splits k
    if (route == K_INNER) part = (size_t)s * ps.M * ps.N * 8;
    if (route == GENERIC && s > 1) part = (size_t)s * ps.M * ps.N * 8;
    *bytes = ((table_bytes(ps) + 255) & ~(size_t)255) + part;
    return PPL_OK;
}

int ppl_contract_pair(const char *subscripts, const int64_t *dims0, const int64_t *dims1, const double *A, const double *B, double *C,
                      double alpha, double beta, void *workspace, size_t workspace_bytes, void *stream_) {
    Parsed ps;
    int rc = parse(subscripts, dims0, dims1, &ps);
    if (rc != PPL_OK) return ppl_fail_code(rc);
    if (!A || !B || !C || (((uintptr_t)A | (uintptr_t)B | (uintptr_t)C) & 7)) return ppl_fail_code(PPL_ERR_INVALID_ARG);
    const ContractDevice *dev = nullptr;
    if ((rc = contract_device(&dev, false)) != PPL_OK) return ppl_fail_code(rc);
    const size_t tb = (table_bytes(ps) + 255) & ~(size_t)255;
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < tb) return ppl_fail_code(PPL_ERR_WORKSPACE_TOO_SMALL);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    const int sms = dev->sms;

    ppl::AxisTables f;
    axis_tables(ps, &f);
    int64_t *tab = reinterpret_cast<int64_t *>(workspace);
    unsigned char *part = reinterpret_cast<unsigned char *>(workspace) + tb;
    ppl::ContractArgs a;
    a.A = A;
    a.B = B;
    a.C = C;
    a.alpha = alpha;
    a.beta = beta;
    table_pointers(ps, tab, &a);
    const bool aligned = (((uintptr_t)A | (uintptr_t)B | (uintptr_t)C) & 15) == 0;
    const Route route = classify(ps, f);
    if (aligned && route == K_OUTER && ps.N * ps.N < ((int64_t)1 << 62))  // no table is read on this route
        return ppl_gemm_kouter_tma(A, B, (int)ps.M, (int)ps.N, (int)ps.K, C, alpha, beta, sms, stream);
    if ((rc = launch_fill(ps, f, tab, sms, stream)) != PPL_OK) return ppl_fail_code(rc);
    if (aligned && route == K_INNER && workspace_bytes - tb >= (size_t)ps.M * ps.N * 8) {
        a.part = reinterpret_cast<double *>(part);
        a.splitk = 1;
        rc = ppl_gemm_kinner_tma(A, B, (int)ps.M, (int)ps.N, (int)ps.K, a.part, workspace_bytes - tb, &a.splitk, sms, stream);
        if (rc != PPL_OK) return rc;
        const int64_t MN = ps.M * ps.N;
        ppl::k_contract_reduce<<<(int)std::min<int64_t>((MN + 255) / 256, (int64_t)sms * 8), 256, 0, stream>>>(a);
        if (cudaGetLastError() != cudaSuccess) return ppl_fail_code(PPL_ERR_CUDA);
        return PPL_OK;
    }
    rc = launch_gather(ps, f, a, part, workspace_bytes - tb, sms, stream);
    return rc == PPL_OK ? PPL_OK : ppl_fail_code(rc);
}

int ppl_contract_pair_noalloc(const char *subscripts, const int64_t *dims0, const int64_t *dims1, const double *A, const double *B,
                              double *C, double alpha, double beta, void *stream_) {
    Parsed ps;
    int rc = parse(subscripts, dims0, dims1, &ps);
    if (rc != PPL_OK) return ppl_fail_code(rc);
    if (!A || !B || !C || (((uintptr_t)A | (uintptr_t)B | (uintptr_t)C) & 7)) return ppl_fail_code(PPL_ERR_INVALID_ARG);
    const size_t tb = (table_bytes(ps) + 255) & ~(size_t)255;
    if (tb > (size_t)PPL_NOALLOC_SCRATCH_BYTES) return ppl_fail_code(PPL_ERR_SCRATCH_LIMIT);
    const ContractDevice *dev = nullptr;
    if ((rc = contract_device(&dev, true)) != PPL_OK) return ppl_fail_code(rc);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);

    ppl::AxisTables f;
    axis_tables(ps, &f);
    int64_t *tab = reinterpret_cast<int64_t *>(dev->scratch);
    if ((rc = launch_fill(ps, f, tab, dev->sms, stream)) != PPL_OK) return ppl_fail_code(rc);
    ppl::ContractArgs a;
    a.A = A;
    a.B = B;
    a.C = C;
    a.alpha = alpha;
    a.beta = beta;
    table_pointers(ps, tab, &a);
    // split-K as ppl_contract_pair picks it for a workspace of PPL_NOALLOC_SCRATCH_BYTES: the partials take what the
    // tables leave, and the factor shrinks (down to 1 = no partials at all) when they would not fit
    rc = launch_gather(ps, f, a, dev->scratch + tb, (size_t)PPL_NOALLOC_SCRATCH_BYTES - tb, dev->sms, stream);
    return rc == PPL_OK ? PPL_OK : ppl_fail_code(rc);
}

}  // extern "C"
