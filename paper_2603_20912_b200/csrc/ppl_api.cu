// ppl_api.cu -- C ABI of libppl (include/ppl.h): planner, W-tile ring, stream orchestration.
// Everything on the data path runs in the kernels of ppl_kernels.cuh; there is no CPU fallback.
#include "../../include/ppl.h"
#include "ppl_kernels.cuh"
#include "ppl_kernels_tma.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

namespace {

thread_local int g_last_error = PPL_OK;

int fail(int code) {
    g_last_error = code;
    return code;
}
#define PPL_CUDA(expr)                                 \
    do {                                               \
        cudaError_t e__ = (expr);                      \
        if (e__ != cudaSuccess) {                      \
            (void)cudaGetLastError();                  \
            return fail(PPL_ERR_CUDA);                 \
        }                                              \
    } while (0)

struct Tile {
    int a0, ta, b0, tb;
    int mirror;
    int splitk, k_per_split;
};

constexpr int MAX_RING = 4;
constexpr double PEAK_FLOPS = 37.2e12;  // nominal FP64 (148 SM x 64 FMA/clk x 2 x 1.965 GHz); planner cost model only
constexpr double HBM_BPS = 6.0e12;      // planner cost model only
constexpr double LAUNCH_S = 4e-6;

}  // namespace

struct ppl_plan_s {
    int o = 0, v = 0, x = 0;
    int sym = PPL_SYM_PAIR;
    int T = 0;            // tile edge (ta = tb = T except at the ragged edge)
    int nblk = 0;
    int ring = 1;
    int vec16 = 0;
    int num_sms = 148;
    int64_t ldw = 0;      // row stride of a W tile (doubles)
    size_t cap = 0;       // workspace cap given by the caller (0 = auto)
    size_t slot_bytes = 0, part_bytes = 0, ws_bytes = 0;
    unsigned char *ws = nullptr;
    double *Wslot[MAX_RING] = {nullptr, nullptr, nullptr, nullptr};
    double *part = nullptr;
    int *flags = nullptr;  // device word for ppl_check_inputs
    std::vector<Tile> tiles;
    cudaStream_t gen = nullptr, host_stream = nullptr;
    cudaEvent_t ev_in = nullptr, ev_ready[MAX_RING] = {}, ev_free[MAX_RING] = {}, ev_gen_done = nullptr;
    // host-path staging buffers (ppl_apply_host)
    double *dL = nullptr, *dT = nullptr, *dR = nullptr;
    double f_step0 = 0, f_step1 = 0;
    int ni1 = 8, bm1 = 128;          // step-1 CTA tile rows = 16*ni1 on the TMA path (128 on the cp.async path)
    int use_tma = 0;                 // 1: persistent TMA/mbarrier kernels (nvirt even); 0: cp.async kernels
    CUtensorMap mapW[MAX_RING];      // W slots as {inner nvirt^2, outer T*T}, built at plan time
};

namespace {

// ------------------------------------------------------------------------------------------
// Planner: the analogue of the paper's memory functions (Table 1) -- but what
// is being sized is the W-tile ring in HBM, not host->device batches.  For a candidate tile edge
// T it estimates the time of one apply from CTA-wave counts of both GEMMs (tile 128x128x16 on
// `sms` SMs), the best split-K per tile shape, and the t2/W streaming traffic.
// ------------------------------------------------------------------------------------------
struct SplitChoice {
    int splitk, k_per_split;
    double seconds;
};

// CTA tile rows of step 1: 16*NI with NI in 5..10 chosen to pad nocc^2 the least (ties: larger tile)
int choose_ni(int M) {
    int best = 8;
    long best_pad = -1;
    for (int ni = 10; ni >= 5; --ni) {
        const long bm = 16 * ni, pad = ((M + bm - 1) / bm) * bm;
        if (best_pad < 0 || pad < best_pad) {
            best_pad = pad;
            best = ni;
        }
    }
    return best;
}

SplitChoice choose_split(int M, int N, int K, int sms, int bm) {
    const int tiles = ((M + bm - 1) / bm) * ((N + ppl::BN - 1) / ppl::BN);
    const int nkt = (K + ppl::BK - 1) / ppl::BK;
    const double tau = 2.0 * bm * ppl::BN * ppl::BK / (PEAK_FLOPS / sms);  // one k-tile on one SM
    SplitChoice best{1, nkt * ppl::BK, 1e300};
    const int smax = std::max(1, std::min(nkt / 8 + 1, 64));
    for (int s = 1; s <= smax; ++s) {
        const int kt_per = (nkt + s - 1) / s;
        const int s_eff = (nkt + kt_per - 1) / kt_per;  // no empty splits
        if (s_eff != s) continue;
        const double waves = std::ceil((double)tiles * s / sms);
        const double t = waves * (kt_per + 6) * tau            // +6: pipeline fill / epilogue
                         + (double)(s + 2) * M * N * 8.0 / HBM_BPS;  // partials written + read by the reduce
        if (t < best.seconds) best = SplitChoice{s, kt_per * ppl::BK, t};
    }
    return best;
}

double step0_seconds(int ta, int tb, int v, int x, int sms) {
    const int tiles = ((ta * v + ppl::BM - 1) / ppl::BM) * ((tb * v + ppl::BN - 1) / ppl::BN);
    const int nkt = (x + ppl::BK - 1) / ppl::BK;
    const double tau = 2.0 * ppl::BM * ppl::BN * ppl::BK / (PEAK_FLOPS / sms);
    return std::ceil((double)tiles / sms) * (nkt + 6) * tau;
}

struct PlanEval {
    double seconds = 1e300;
    size_t slot_bytes = 0, part_bytes = 0;
};

PlanEval evaluate(int o, int v, int x, int T, int sym, int sms, int bm1) {
    PlanEval ev;
    const int nblk = (v + T - 1) / T;
    const int64_t vv = (int64_t)v * v;
    const int M = o * o;
    const double t2_bytes = (double)M * vv * 8.0;
    double total = 0;
    size_t part_max = 0;
    // distinct tile shapes: (T,T), (T,r), (r,T), (r,r) with r = ragged edge
    const int r = v - (nblk - 1) * T;
    auto count = [&](bool a_edge, bool b_edge) -> int64_t {
        // number of executed tiles with the given edge flags
        const int na = a_edge ? 1 : nblk - 1, nb = b_edge ? 1 : nblk - 1;
        if (!sym) return (int64_t)na * nb;
        // tiles with ablock <= bblock
        if (a_edge && b_edge) return 1;
        if (a_edge && !b_edge) return 0;                  // a = last block, b < last: a > b
        if (!a_edge && b_edge) return nblk - 1;           // every a-block below the last pairs with the last
        return (int64_t)(nblk - 1) * nblk / 2;            // interior a<=b
    };
    for (int ae = 0; ae < 2; ++ae)
        for (int be = 0; be < 2; ++be) {
            const int64_t cnt = count(ae, be);
            if (cnt == 0) continue;
            const int ta = ae ? r : T, tb = be ? r : T;
            const int N = ta * tb;
            const SplitChoice sc = choose_split(M, N, (int)std::min<int64_t>(vv, INT32_MAX), sms, bm1);
            const double compute = step0_seconds(ta, tb, v, x, sms) + sc.seconds;
            const double dram = (t2_bytes + 2.0 * N * vv * 8.0) / HBM_BPS;
            total += cnt * (std::max(compute, dram) + 3 * LAUNCH_S);
            part_max = std::max(part_max, (size_t)sc.splitk * M * N * 8);
        }
    ev.seconds = total;
    ev.slot_bytes = (size_t)T * T * vv * 8;
    ev.part_bytes = part_max;
    return ev;
}

int build_tiles(ppl_plan_s *p) {
    p->tiles.clear();
    p->f_step0 = p->f_step1 = 0;
    const int T = p->T, v = p->v;
    const int64_t vv = (int64_t)v * v;
    for (int ab = 0; ab < p->nblk; ++ab)
        for (int bb = (p->sym == PPL_SYM_PAIR ? ab : 0); bb < p->nblk; ++bb) {
            Tile t;
            t.a0 = ab * T;
            t.ta = std::min(T, v - t.a0);
            t.b0 = bb * T;
            t.tb = std::min(T, v - t.b0);
            t.mirror = (p->sym == PPL_SYM_PAIR && ab != bb) ? 1 : 0;
            const SplitChoice sc = choose_split(p->o * p->o, t.ta * t.tb, (int)vv, p->num_sms, p->bm1);
            t.splitk = sc.splitk;
            t.k_per_split = sc.k_per_split;
            if ((size_t)t.splitk * p->o * p->o * t.ta * t.tb * 8 > p->part_bytes) return PPL_ERR_WORKSPACE_TOO_SMALL;
            p->tiles.push_back(t);
            p->f_step0 += 2.0 * p->x * (double)t.ta * t.tb * (double)vv;
            p->f_step1 += 2.0 * p->o * p->o * (double)t.ta * t.tb * (double)vv;
        }
    return PPL_OK;
}

void free_plan(ppl_plan_s *p) {
    if (!p) return;
    if (p->gen) {
        cudaStreamSynchronize(p->gen);
        cudaStreamDestroy(p->gen);
    }
    if (p->host_stream) {
        cudaStreamSynchronize(p->host_stream);
        cudaStreamDestroy(p->host_stream);
    }
    if (p->ev_in) cudaEventDestroy(p->ev_in);
    if (p->ev_gen_done) cudaEventDestroy(p->ev_gen_done);
    for (int i = 0; i < MAX_RING; ++i) {
        if (p->ev_ready[i]) cudaEventDestroy(p->ev_ready[i]);
        if (p->ev_free[i]) cudaEventDestroy(p->ev_free[i]);
    }
    if (p->ws) cudaFree(p->ws);
    if (p->flags) cudaFree(p->flags);
    if (p->dL) cudaFree(p->dL);
    if (p->dT) cudaFree(p->dT);
    if (p->dR) cudaFree(p->dR);
    delete p;
}

bool g_attr_set = false;
int set_kernel_attrs() {
    if (g_attr_set) return PPL_OK;
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_MN));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_MN));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_K));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_K));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_TMA));
#define PPL_ATTR_NI(NI) \
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1_tma<NI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::Step1Cfg<NI>::SMEM));
    PPL_ATTR_NI(5) PPL_ATTR_NI(6) PPL_ATTR_NI(7) PPL_ATTR_NI(8) PPL_ATTR_NI(9) PPL_ATTR_NI(10)
#undef PPL_ATTR_NI
    g_attr_set = true;
    return PPL_OK;
}

int launch_step0(const ppl_plan_s *p, const Tile &t, const double *L, double *W, bool vec16, cudaStream_t s) {
    ppl::Step0Args a;
    a.A = L + (int64_t)t.a0 * p->v;
    a.B = L + (int64_t)t.b0 * p->v;
    a.ld = (int64_t)p->v * p->v;
    a.M = t.ta * p->v;
    a.N = t.tb * p->v;
    a.K = p->x;
    a.v = p->v;
    a.tb = t.tb;
    a.W = W;
    a.ldw = p->ldw;
    const int grid = ((a.M + ppl::BM - 1) / ppl::BM) * ((a.N + ppl::BN - 1) / ppl::BN);
    if (vec16)
        ppl::k_step0<2><<<grid, ppl::NTHREADS, ppl::SMEM_MN, s>>>(a);
    else
        ppl::k_step0<1><<<grid, ppl::NTHREADS, ppl::SMEM_MN, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int launch_step1(const ppl_plan_s *p, const Tile &t, const double *t2, const double *W, bool vec16, cudaStream_t s) {
    ppl::Step1Args a;
    a.A = t2;
    a.B = W;
    a.lda = (int64_t)p->v * p->v;
    a.ldb = p->ldw;
    a.M = p->o * p->o;
    a.N = t.ta * t.tb;
    a.K = p->v * p->v;
    a.k_per_split = t.k_per_split;
    a.part = p->part;
    dim3 grid(((a.M + ppl::BM - 1) / ppl::BM) * ((a.N + ppl::BN - 1) / ppl::BN), t.splitk);
    if (vec16)
        ppl::k_step1<2><<<grid, ppl::NTHREADS, ppl::SMEM_K, s>>>(a);
    else
        ppl::k_step1<1><<<grid, ppl::NTHREADS, ppl::SMEM_K, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int launch_reduce(const ppl_plan_s *p, const Tile &t, double *R, cudaStream_t s) {
    ppl::ReduceArgs a;
    a.part = p->part;
    a.splitk = t.splitk;
    a.M = p->o * p->o;
    a.N = t.ta * t.tb;
    a.o = p->o;
    a.v = p->v;
    a.tb = t.tb;
    a.a0 = t.a0;
    a.b0 = t.b0;
    a.mirror = t.mirror;
    a.R = R;
    const int64_t MN = (int64_t)a.M * a.N;
    const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
    ppl::k_reduce<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}


// ---- TMA tensor maps (driver entry point fetched through the runtime: no libcuda link) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
        else
            (void)cudaGetLastError();
    }
    return fn;
}
// 2-D FP64 tensor {inner (contiguous), outer} with row stride `row_bytes`, box {box_inner, box_outer}, 128B swizzle
int make_map_2d(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t row_bytes, uint32_t box_inner,
                uint32_t box_outer) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return PPL_ERR_CUDA;
    const cuuint64_t gdim[2] = {inner, outer};
    const cuuint64_t gstride[1] = {row_bytes};
    const cuuint32_t box[2] = {box_inner, box_outer};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? PPL_OK : PPL_ERR_CUDA;
}

int launch_step0_tma(const ppl_plan_s *p, const Tile &t, const CUtensorMap &mapL, double *W, cudaStream_t s) {
    ppl::Step0TmaArgs a;
    a.a0v = t.a0 * p->v;
    a.b0v = t.b0 * p->v;
    a.M = t.ta * p->v;
    a.N = t.tb * p->v;
    a.K = p->x;
    a.v = p->v;
    a.tb = t.tb;
    a.W = W;
    a.ldw = p->ldw;
    const int items = ((a.M + ppl::BM - 1) / ppl::BM) * ((a.N + ppl::BN - 1) / ppl::BN);
    ppl::k_step0_tma<<<std::min(items, p->num_sms), ppl::TMA_THREADS, ppl::SMEM_TMA, s>>>(mapL, a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int launch_step1_tma(const ppl_plan_s *p, const Tile &t, const CUtensorMap &mapT, const CUtensorMap &mapW, cudaStream_t s) {
    ppl::Step1TmaArgs a;
    a.M = p->o * p->o;
    a.N = t.ta * t.tb;
    a.K = p->v * p->v;
    a.k_per_split = t.k_per_split;
    a.splitk = t.splitk;
    a.part = p->part;
    const int items = ((a.M + p->bm1 - 1) / p->bm1) * ((a.N + ppl::BN - 1) / ppl::BN) * t.splitk;
    const int grid = std::min(items, p->num_sms);
    switch (p->ni1) {
#define PPL_LAUNCH_NI(NI)                                                                                        \
    case NI:                                                                                                     \
        ppl::k_step1_tma<NI><<<grid, ppl::TMA_THREADS, ppl::Step1Cfg<NI>::SMEM, s>>>(mapT, mapW, a);           \
        break;
        PPL_LAUNCH_NI(5) PPL_LAUNCH_NI(6) PPL_LAUNCH_NI(7) PPL_LAUNCH_NI(8) PPL_LAUNCH_NI(9) PPL_LAUNCH_NI(10)
#undef PPL_LAUNCH_NI
        default: return fail(PPL_ERR_INVALID_ARG);
    }
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

struct ApplyMaps {
    CUtensorMap L, T;
};
int make_apply_maps(const ppl_plan_s *p, const double *L, const double *t2, ApplyMaps *m) {
    const uint64_t vv = (uint64_t)p->v * p->v;
    int rc = make_map_2d(&m->L, L, vv, (uint64_t)p->x, vv * 8, 16, ppl::BK);
    if (rc == PPL_OK) rc = make_map_2d(&m->T, t2, vv, (uint64_t)p->o * p->o, vv * 8, ppl::BK, (uint32_t)p->bm1);
    return rc;
}

int check_ptrs(const ppl_plan_s *p, const double *L, const double *t2, const double *R, bool *vec16) {
    if (!p || !L || !t2 || !R) return PPL_ERR_INVALID_ARG;
    const uintptr_t all = (uintptr_t)L | (uintptr_t)t2 | (uintptr_t)R;
    if (all & 7) return PPL_ERR_INVALID_ARG;
    *vec16 = p->vec16 && ((all & 15) == 0);
    return PPL_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

int ppl_last_error(void) { return g_last_error; }

const char *ppl_error_string(int code) {
    switch (code) {
        case PPL_OK: return "ok";
        case PPL_ERR_INVALID_ARG: return "invalid argument";
        case PPL_ERR_WORKSPACE_TOO_SMALL: return "workspace_bytes below the minimum plan";
        case PPL_ERR_ALLOC: return "allocation failed";
        case PPL_ERR_CUDA: return "CUDA runtime error";
        case PPL_ERR_UNSUPPORTED_DEVICE: return "no CUDA device of compute capability 10.x (no fallback path exists)";
        case PPL_ERR_PRECONDITION: return "input violates a symmetry the plan relies on";
        default: return "unknown error";
    }
}

ppl_plan_t *ppl_plan(int nocc, int nvirt, int nchol, size_t workspace_bytes) {
    if (nocc < 1 || nvirt < 1 || nchol < 1 || (int64_t)nvirt * nvirt > INT32_MAX / 2 ||
        (int64_t)nocc * nocc > INT32_MAX / 2) {
        fail(PPL_ERR_INVALID_ARG);
        return nullptr;
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        fail(PPL_ERR_UNSUPPORTED_DEVICE);
        return nullptr;
    }
    if (prop.major != 10) {
        fail(PPL_ERR_UNSUPPORTED_DEVICE);
        return nullptr;
    }
    ppl_plan_s *p = new (std::nothrow) ppl_plan_s();
    if (!p) {
        fail(PPL_ERR_ALLOC);
        return nullptr;
    }
    p->o = nocc;
    p->v = nvirt;
    p->x = nchol;
    p->num_sms = prop.multiProcessorCount;
    p->vec16 = (nvirt % 2 == 0) ? 1 : 0;
    p->ldw = (int64_t)nvirt * nvirt;
    p->cap = workspace_bytes;

    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) {
        (void)cudaGetLastError();
        free_plan(p);
        fail(PPL_ERR_CUDA);
        return nullptr;
    }
    const size_t auto_cap = (size_t)(0.9 * (double)free_b);
    const size_t cap = workspace_bytes ? std::min(workspace_bytes, auto_cap) : auto_cap;

    const char *envk = getenv("PPL_KERNELS");  // debug override: "cpasync" forces the non-TMA kernels
    p->use_tma = p->vec16 && !(envk && strcmp(envk, "cpasync") == 0) && get_encode() != nullptr;
    if (p->use_tma) {
        const char *envni = getenv("PPL_NI");  // debug override of the step-1 tile height
        p->ni1 = (envni && atoi(envni) >= 5 && atoi(envni) <= 10) ? atoi(envni) : choose_ni(nocc * nocc);
        p->bm1 = 16 * p->ni1;
    }
    // choose the tile edge T (and ring depth) that minimises the estimated apply time under the cap
    const char *envT = getenv("PPL_TILE");  // debug override
    double best_t = 1e300;
    int best_T = 0, best_ring = 1;
    PlanEval best_ev;
    for (int T = nvirt; T >= 1; --T) {
        if (envT && atoi(envT) > 0 && T != std::min(atoi(envT), nvirt)) continue;
        // only edges that tile v evenly or nearly so (ragged edge at least T/2), to keep edge tiles efficient
        const int nblk = (nvirt + T - 1) / T;
        const int r = nvirt - (nblk - 1) * T;
        if (!envT && nblk > 1 && 2 * r < T) continue;
        const PlanEval ev = evaluate(nocc, nvirt, nchol, T, PPL_SYM_PAIR, p->num_sms, p->bm1);
        // the same plan must also serve PPL_SYM_NONE (same shapes), so part/slot sizes are identical
        int ring = 0;
        for (int rg = std::min(3, MAX_RING); rg >= 1; --rg)
            if (rg * ev.slot_bytes + ev.part_bytes + 256 <= cap) {
                ring = rg;
                break;
            }
        if (ring == 0) continue;
        const int ntiles = nblk * (nblk + 1) / 2;
        ring = std::min(ring, std::max(1, ntiles));
        const double t = ev.seconds * (ring >= 2 ? 1.0 : 1.03);
        if (t < best_t) {
            best_t = t;
            best_T = T;
            best_ring = ring;
            best_ev = ev;
        }
    }
    if (best_T == 0) {
        free_plan(p);
        fail(PPL_ERR_WORKSPACE_TOO_SMALL);
        return nullptr;
    }
    p->T = best_T;
    p->nblk = (nvirt + best_T - 1) / best_T;
    p->ring = best_ring;
    p->slot_bytes = (best_ev.slot_bytes + 255) & ~(size_t)255;
    p->part_bytes = (best_ev.part_bytes + 255) & ~(size_t)255;
    p->ws_bytes = p->ring * p->slot_bytes + p->part_bytes;
    if (cudaMalloc(&p->ws, p->ws_bytes) != cudaSuccess || cudaMalloc(&p->flags, sizeof(int)) != cudaSuccess) {
        (void)cudaGetLastError();
        free_plan(p);
        fail(PPL_ERR_ALLOC);
        return nullptr;
    }
    for (int i = 0; i < p->ring; ++i) p->Wslot[i] = reinterpret_cast<double *>(p->ws + (size_t)i * p->slot_bytes);
    p->part = reinterpret_cast<double *>(p->ws + (size_t)p->ring * p->slot_bytes);

    bool ok = cudaStreamCreateWithFlags(&p->gen, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&p->host_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&p->ev_in, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&p->ev_gen_done, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < MAX_RING && ok; ++i) {
        ok = ok && cudaEventCreateWithFlags(&p->ev_ready[i], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&p->ev_free[i], cudaEventDisableTiming) == cudaSuccess;
    }
    if (!ok || set_kernel_attrs() != PPL_OK) {
        (void)cudaGetLastError();
        free_plan(p);
        fail(PPL_ERR_CUDA);
        return nullptr;
    }
    if (p->use_tma) {
        const uint64_t vv = (uint64_t)nvirt * nvirt;
        for (int i = 0; i < p->ring; ++i)
            if (make_map_2d(&p->mapW[i], p->Wslot[i], vv, (uint64_t)p->T * p->T, (uint64_t)p->ldw * 8, ppl::BK, ppl::BN) != PPL_OK) {
                p->use_tma = 0;
                break;
            }
    }
    p->sym = PPL_SYM_PAIR;
    const int rc = build_tiles(p);
    if (rc != PPL_OK) {
        free_plan(p);
        fail(rc);
        return nullptr;
    }
    return p;
}

int ppl_plan_set_symmetry(ppl_plan_t *p, int mode) {
    if (!p || (mode != PPL_SYM_NONE && mode != PPL_SYM_PAIR)) return fail(PPL_ERR_INVALID_ARG);
    p->sym = mode;
    const int rc = build_tiles(p);
    return rc == PPL_OK ? PPL_OK : fail(rc);
}

int ppl_plan_info(const ppl_plan_t *p, ppl_info_t *out) {
    if (!p || !out) return fail(PPL_ERR_INVALID_ARG);
    memset(out, 0, sizeof(*out));
    out->nocc = p->o;
    out->nvirt = p->v;
    out->nchol = p->x;
    out->symmetry = p->sym;
    out->ta = out->tb = p->T;
    out->n_ablocks = out->n_bblocks = p->nblk;
    out->n_tiles = (int)p->tiles.size();
    out->ring = p->ring;
    out->splitk = p->tiles.empty() ? 0 : p->tiles[0].splitk;
    out->vec16 = p->vec16;
    out->launches_per_apply = 3 * (int)p->tiles.size();
    out->step1_tile_m = p->bm1;
    out->workspace_bytes = p->ws_bytes;
    const double v4 = std::pow((double)p->v, 4);
    out->flops_nominal = 2.0 * p->x * v4 + 2.0 * p->o * p->o * v4;
    out->flops_step0 = p->f_step0;
    out->flops_step1 = p->f_step1;
    out->flops_executed = p->f_step0 + p->f_step1;
    return PPL_OK;
}

int ppl_apply(ppl_plan_t *p, const double *L, const double *t2, double *R, void *stream_) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, t2, R, &vec16);
    if (rc != PPL_OK) return fail(rc);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    const int ntiles = (int)p->tiles.size();
    const bool tma = p->use_tma && vec16;
    ApplyMaps maps;
    if (tma && (rc = make_apply_maps(p, L, t2, &maps)) != PPL_OK) return fail(rc);
    const bool two_streams = p->ring >= 2 && ntiles >= 2;
    cudaStream_t gen = two_streams ? p->gen : stream;

    if (two_streams) {  // fork: the producer stream starts after prior work on `stream`
        PPL_CUDA(cudaEventRecord(p->ev_in, stream));
        PPL_CUDA(cudaStreamWaitEvent(gen, p->ev_in, 0));
    }
    for (int k = 0; k < ntiles; ++k) {
        const Tile &t = p->tiles[k];
        const int slot = k % p->ring;
        if (two_streams && k >= p->ring) PPL_CUDA(cudaStreamWaitEvent(gen, p->ev_free[slot], 0));
        rc = tma ? launch_step0_tma(p, t, maps.L, p->Wslot[slot], gen) : launch_step0(p, t, L, p->Wslot[slot], vec16, gen);
        if (rc != PPL_OK) return rc;
        if (two_streams) {
            PPL_CUDA(cudaEventRecord(p->ev_ready[slot], gen));
            PPL_CUDA(cudaStreamWaitEvent(stream, p->ev_ready[slot], 0));
        }
        rc = tma ? launch_step1_tma(p, t, maps.T, p->mapW[slot], stream) : launch_step1(p, t, t2, p->Wslot[slot], vec16, stream);
        if (rc != PPL_OK) return rc;
        if (two_streams) PPL_CUDA(cudaEventRecord(p->ev_free[slot], stream));
        if ((rc = launch_reduce(p, t, R, stream)) != PPL_OK) return rc;
    }
    // join: every producer launch is followed by a consumer wait on `stream`, so `stream` already
    // depends on all work of `gen`.
    return PPL_OK;
}

int ppl_apply_profiled(ppl_plan_t *p, const double *L, const double *t2, double *R, void *stream_, ppl_times_t *times) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, t2, R, &vec16);
    if (rc != PPL_OK || !times) return fail(rc != PPL_OK ? rc : PPL_ERR_INVALID_ARG);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    memset(times, 0, sizeof(*times));
    const int ntiles = (int)p->tiles.size();
    const bool tma = p->use_tma && vec16;
    ApplyMaps maps;
    if (tma && (rc = make_apply_maps(p, L, t2, &maps)) != PPL_OK) return fail(rc);
    std::vector<cudaEvent_t> ev(3 * (size_t)ntiles + 1);
    for (auto &e : ev) PPL_CUDA(cudaEventCreate(&e));
    PPL_CUDA(cudaEventRecord(ev[0], stream));
    for (int k = 0; k < ntiles && rc == PPL_OK; ++k) {
        const Tile &t = p->tiles[k];
        rc = tma ? launch_step0_tma(p, t, maps.L, p->Wslot[0], stream) : launch_step0(p, t, L, p->Wslot[0], vec16, stream);
        cudaEventRecord(ev[3 * k + 1], stream);
        if (rc == PPL_OK)
            rc = tma ? launch_step1_tma(p, t, maps.T, p->mapW[0], stream) : launch_step1(p, t, t2, p->Wslot[0], vec16, stream);
        cudaEventRecord(ev[3 * k + 2], stream);
        if (rc == PPL_OK) rc = launch_reduce(p, t, R, stream);
        cudaEventRecord(ev[3 * k + 3], stream);
    }
    cudaError_t e = cudaStreamSynchronize(stream);
    if (rc == PPL_OK && e == cudaSuccess) {
        for (int k = 0; k < ntiles; ++k) {
            float a = 0, b = 0, c = 0;
            cudaEventElapsedTime(&a, ev[3 * k], ev[3 * k + 1]);
            cudaEventElapsedTime(&b, ev[3 * k + 1], ev[3 * k + 2]);
            cudaEventElapsedTime(&c, ev[3 * k + 2], ev[3 * k + 3]);
            times->step0_ms += a;
            times->step1_ms += b;
            times->reduce_ms += c;
        }
        cudaEventElapsedTime(&times->total_ms, ev[0], ev[3 * (size_t)ntiles]);
        times->n_step0 = times->n_step1 = times->n_reduce = ntiles;
    }
    for (auto &x : ev) cudaEventDestroy(x);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(PPL_ERR_CUDA);
    }
    return rc;
}

int ppl_apply_host(ppl_plan_t *p, const double *Lh, const double *t2h, double *Rh, uint64_t *h2d, uint64_t *d2h) {
    if (!p || !Lh || !t2h || !Rh) return fail(PPL_ERR_INVALID_ARG);
    const size_t nL = (size_t)p->x * p->v * p->v * 8, nT = (size_t)p->o * p->o * p->v * p->v * 8;
    if (!p->dL) {
        if (cudaMalloc(&p->dL, nL) != cudaSuccess || cudaMalloc(&p->dT, nT) != cudaSuccess ||
            cudaMalloc(&p->dR, nT) != cudaSuccess) {
            (void)cudaGetLastError();
            if (p->dL) cudaFree(p->dL);
            if (p->dT) cudaFree(p->dT);
            if (p->dR) cudaFree(p->dR);
            p->dL = p->dT = p->dR = nullptr;
            return fail(PPL_ERR_ALLOC);
        }
    }
    cudaStream_t s = p->host_stream;
    PPL_CUDA(cudaMemcpyAsync(p->dL, Lh, nL, cudaMemcpyHostToDevice, s));
    PPL_CUDA(cudaMemcpyAsync(p->dT, t2h, nT, cudaMemcpyHostToDevice, s));
    PPL_CUDA(cudaMemcpyAsync(p->dR, Rh, nT, cudaMemcpyHostToDevice, s));
    int rc = ppl_apply(p, p->dL, p->dT, p->dR, s);
    if (rc == PPL_OK) {
        cudaError_t e = cudaMemcpyAsync(Rh, p->dR, nT, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            rc = fail(PPL_ERR_CUDA);
        }
    }
    if (h2d) *h2d = (uint64_t)nL + 2 * (uint64_t)nT;
    if (d2h) *d2h = (uint64_t)nT;
    return rc;
}

int ppl_check_inputs(ppl_plan_t *p, const double *L, const double *t2, void *stream_, int *flags) {
    if (!p || !L || !t2) return fail(PPL_ERR_INVALID_ARG);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    PPL_CUDA(cudaMemsetAsync(p->flags, 0, sizeof(int), stream));
    ppl::k_check_inputs<<<p->num_sms * 8, 256, 0, stream>>>(L, t2, p->o, p->v, p->x, p->flags);
    PPL_CUDA(cudaGetLastError());
    int h = 0;
    PPL_CUDA(cudaMemcpyAsync(&h, p->flags, sizeof(int), cudaMemcpyDeviceToHost, stream));
    PPL_CUDA(cudaStreamSynchronize(stream));
    if (flags) *flags = h;
    if ((h & 2) && p->sym == PPL_SYM_PAIR) return fail(PPL_ERR_PRECONDITION);
    return PPL_OK;
}

int ppl_destroy(ppl_plan_t *p) {
    if (!p) return PPL_OK;
    free_plan(p);
    return PPL_OK;
}

int ppl_probe_fp64_peak(double *tflops, int reps, double ms_target) {
    if (!tflops || reps < 1) return fail(PPL_ERR_INVALID_ARG);
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) {
        (void)cudaGetLastError();
        return fail(PPL_ERR_UNSUPPORTED_DEVICE);
    }
    double *out = nullptr;
    PPL_CUDA(cudaMalloc(&out, 64));
    cudaEvent_t e0, e1;
    PPL_CUDA(cudaEventCreate(&e0));
    PPL_CUDA(cudaEventCreate(&e1));
    const int sms = prop.multiProcessorCount, threads = 512;
    // 8 DMMA per iteration per warp, 512 flop each
    const double flop_per_iter = 512.0 * 8 * (threads / 32) * sms;
    int iters = (int)std::max(1024.0, ms_target * 1e-3 * PEAK_FLOPS / flop_per_iter);
    double best = 0;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0, 0);
        ppl::k_probe_dmma<<<sms, threads>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            (void)cudaGetLastError();
            cudaFree(out);
            return fail(PPL_ERR_CUDA);
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0) best = std::max(best, flop_per_iter * iters / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = best;
    return PPL_OK;
}

// test hook: C(8x8) = A(8x4) B(4x8) through one DMMA with the fragment layout the kernels assume
int ppl_debug_dmma_layout(const double *A_dev, const double *B_dev, double *C_dev) {
    if (!A_dev || !B_dev || !C_dev) return fail(PPL_ERR_INVALID_ARG);
    ppl::k_dmma_layout<<<1, 32>>>(A_dev, B_dev, C_dev);
    PPL_CUDA(cudaGetLastError());
    PPL_CUDA(cudaDeviceSynchronize());
    return PPL_OK;
}

}  // extern "C"
