// ppl_api.cu -- C ABI of libppl (include/ppl.h): device allocation, launches, W-tile ring, stream orchestration, host
// streaming, probes.  The planner is ppl_plan.cpp (host only).  Everything on the data path runs in the kernels of
// ppl_kernels*.cuh; there is no CPU fallback.
#include "../../include/ppl.h"
#include "ppl_plan.h"
#include "ppl_launch.h"
#include "ppl_kernels.cuh"
#include "ppl_kernels_tma.cuh"
#include "ppl_kernels_full.cuh"
#include "ppl_kernels_small.cuh"

#include <atomic>
#include <initializer_list>
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace pplh;

namespace {
#define PPL_CUDA(expr)                                 \
    do {                                               \
        cudaError_t e__ = (expr);                      \
        if (e__ != cudaSuccess) {                      \
            (void)cudaGetLastError();                  \
            return fail(PPL_ERR_CUDA);                 \
        }                                              \
    } while (0)
}  // namespace

namespace {

// per-apply verification of the symmetry preconditions (PPL_OPT_VERIFY_INPUTS; defined next to ppl_check_inputs)
int verify_harvest(ppl_plan_s *p, int *flags_out, bool wait_all = true);
int verify_begin(ppl_plan_s *p, const double *L, const double *t2, int t2_layout, cudaStream_t stream);

void free_plan(ppl_plan_s *p) {
    if (!p) return;
    // applies (plain launches on the caller's stream, or a graph launch) may still be in flight on streams the plan
    // does not own: wait for the device before the workspace goes away
    const bool owns_device = p->ws || p->fws || p->vflags_host || p->gen || p->gexec;  // not so for ppl_plan_dry or a plan that failed early
    if (!p->dry && owns_device && cudaDeviceSynchronize() != cudaSuccess) (void)cudaGetLastError();
    if (p->gen) {
        cudaStreamSynchronize(p->gen);
        cudaStreamDestroy(p->gen);
    }
    if (p->host_stream) {
        cudaStreamSynchronize(p->host_stream);
        cudaStreamDestroy(p->host_stream);
    }
    if (p->ev_in) cudaEventDestroy(p->ev_in);
    if (p->gexec) cudaGraphExecDestroy(p->gexec);
    if (p->gcap) cudaStreamDestroy(p->gcap);
    if (p->hs2) {
        cudaStreamSynchronize(p->hs2);
        cudaStreamDestroy(p->hs2);
    }
    if (p->ev_tau) cudaEventDestroy(p->ev_tau);
    if (p->ev_done) cudaEventDestroy(p->ev_done);
    for (int i = 0; i < 4; ++i)
        if (p->fs[i]) {
            cudaStreamSynchronize(p->fs[i]);
            cudaStreamDestroy(p->fs[i]);
        }
    if (p->fs0) {
        cudaStreamSynchronize(p->fs0);
        cudaStreamDestroy(p->fs0);
    }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    for (int s = 0; s < 2; ++s) {
        if (p->ev_s0[s]) cudaEventDestroy(p->ev_s0[s]);
        if (p->ev_xfree[s]) cudaEventDestroy(p->ev_xfree[s]);
    }
    for (int s = 0; s < 2; ++s) {
        if (p->ev_fold[s]) cudaEventDestroy(p->ev_fold[s]);
        for (int i = 0; i < 4; ++i)
            if (p->evg[s][i]) cudaEventDestroy(p->evg[s][i]);
    }
    for (int i = 0; i < MAX_RING; ++i) {
        if (p->ev_ready[i]) cudaEventDestroy(p->ev_ready[i]);
        if (p->ev_free[i]) cudaEventDestroy(p->ev_free[i]);
    }
    if (p->ws) cudaFree(p->ws);
    if (p->fws) cudaFree(p->fws);
    if (p->small_Lp) cudaFree(p->small_Lp);
    if (p->small_tp) cudaFree(p->small_tp);
    if (p->vflags_host) cudaFreeHost(p->vflags_host);
    if (p->vdone_dev) cudaFree(p->vdone_dev);
    if (p->ev_verify) cudaEventDestroy(p->ev_verify);
    for (cudaEvent_t e : {p->ev_vq[0], p->ev_vq[1]})
        if (e) cudaEventDestroy(e);
    if (p->tperm) cudaFree(p->tperm);
    if (p->dL) cudaFree(p->dL);
    if (p->dT) cudaFree(p->dT);
    if (p->dR) cudaFree(p->dR);
    for (int i = 0; i < 2; ++i)
        if (p->hstage[i]) cudaFree(p->hstage[i]);
    {
        ppl_plan_s::HostStream &h = p->hsn;
        for (cudaStream_t st : {h.in, h.out})
            if (st) {
                cudaStreamSynchronize(st);
                cudaStreamDestroy(st);
            }
        for (int i = 0; i < 2; ++i) {
            if (h.pa[i]) cudaFree(h.pa[i]);
            if (h.rs[i]) cudaFree(h.rs[i]);
            for (cudaEvent_t e : {h.ev_pa[i], h.ev_pafree[i], h.ev_rsin[i], h.ev_rsdone[i], h.ev_rsfree[i], h.ev_chunk[i]})
                if (e) cudaEventDestroy(e);
        }
        for (int i = 0; i < MAX_RING; ++i) {
            if (h.pb[i]) cudaFree(h.pb[i]);
            for (cudaEvent_t e : {h.ev_pb[i], h.ev_pbfree[i]})
                if (e) cudaEventDestroy(e);
        }
        for (cudaEvent_t e : {h.ev_t2, h.ev_fork})
            if (e) cudaEventDestroy(e);
    }
    delete p;
}

std::atomic<bool> g_attr_set[64];  // per device: function attributes belong to the device's context
int set_kernel_attrs() {
    int dev = 0;
    PPL_CUDA(cudaGetDevice(&dev));
    const bool known = dev >= 0 && dev < 64;
    if (known && g_attr_set[dev].load()) return PPL_OK;
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_MN));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_MN));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_K));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_K));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_TMA));
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step0_slab, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::SMEM_TMA));
#define PPL_ATTR_NI(NI)                                                                                                                \
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1_tma<NI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::Step1Cfg<NI>::SMEM)); \
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_step1t_tma<NI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ppl::Step1Cfg<NI>::SMEM));
    PPL_ATTR_NI(1) PPL_ATTR_NI(2) PPL_ATTR_NI(3) PPL_ATTR_NI(4) PPL_ATTR_NI(5) PPL_ATTR_NI(6) PPL_ATTR_NI(7) PPL_ATTR_NI(8) PPL_ATTR_NI(9) PPL_ATTR_NI(10)
#undef PPL_ATTR_NI
#define PPL_ATTR_SMALL(NB) \
    PPL_CUDA(cudaFuncSetAttribute(ppl::k_small_fused<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    PPL_ATTR_SMALL(1) PPL_ATTR_SMALL(2) PPL_ATTR_SMALL(3) PPL_ATTR_SMALL(4) PPL_ATTR_SMALL(5) PPL_ATTR_SMALL(6) PPL_ATTR_SMALL(7)
#undef PPL_ATTR_SMALL
    if (known) g_attr_set[dev].store(true);
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
// 2-D FP64 tensor {inner (contiguous), outer} with row stride `row_bytes`, box {box_inner, box_outer}, 128B swizzle;
// out-of-bounds elements of a box are filled with zeros (tile edges, k tails)
int make_map_2d(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t row_bytes, uint32_t box_inner,
                uint32_t box_outer, bool promo128 = false) {
    EncodeTiledFn enc = get_encode();
    if (!enc || inner == 0 || outer == 0) return PPL_ERR_CUDA;
    const cuuint64_t gdim[2] = {inner, outer};
    const cuuint64_t gstride[1] = {row_bytes};
    const cuuint32_t box[2] = {box_inner, box_outer};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           promo128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? PPL_OK : PPL_ERR_CUDA;
}

// ---- launches ----
int launch_step0(const ppl_plan_s *p, const Tile &t, const double *L, const CUtensorMap *mapL, double *W, bool vec16,
                 cudaStream_t s) {
    const int M = t.ta * p->v, N = t.tb * p->v;
    const int items = ((M + ppl::BM - 1) / ppl::BM) * ((N + ppl::BN - 1) / ppl::BN);
    if (mapL) {
        ppl::Step0TmaArgs a;
        a.a0v = t.a0 * p->v;
        a.b0v = t.b0 * p->v;
        a.M = M;
        a.N = N;
        a.K = p->x;
        a.v = p->v;
        a.tb = t.tb;
        a.W = W;
        a.ldw = p->vv;
        ppl::k_step0_tma<<<std::min(items, p->num_sms), ppl::TMA_THREADS, ppl::SMEM_TMA, s>>>(*mapL, *mapL, a);
    } else {
        ppl::Step0Args a;
        a.A = L + (int64_t)t.a0 * p->v;
        a.B = L + (int64_t)t.b0 * p->v;
        a.ld = p->vv;
        a.M = M;
        a.N = N;
        a.K = p->x;
        a.v = p->v;
        a.tb = t.tb;
        a.W = W;
        a.ldw = p->vv;
        if (vec16)
            ppl::k_step0<2><<<items, ppl::NTHREADS, ppl::SMEM_MN, s>>>(a);
        else
            ppl::k_step0<1><<<items, ppl::NTHREADS, ppl::SMEM_MN, s>>>(a);
    }
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// One step-1 GEMM: part[z][M][N] = sum_{k in split z} A[m][k] B[n][k]; A is lda-strided, B ldb-strided.
// With maps: the persistent TMA kernel with CTA tile (16*ni) x 128; without: the cp.async kernel.
int launch_step1(const ppl_plan_s *p, const CUtensorMap *mapA, const CUtensorMap *mapB, const MGeom &mg, const double *A, int64_t lda,
                 const double *B, int64_t ldb, int M, int N, int64_t K, const SplitChoice &sc, double *part, bool vec16,
                 cudaStream_t s, int k0 = 0) {
    if (M <= 0 || N <= 0 || K - k0 <= 0) return PPL_OK;
    if (k0 != 0 && !(mapA && mapB)) return fail(PPL_ERR_INVALID_ARG);
    if (mapA && mapB) {
        ppl::Step1TmaArgs a;
        a.M = M;
        a.N = N;
        a.K = (int)K;
        a.k0 = k0;
        a.k_per_split = sc.k_per_split;
        a.splitk = sc.splitk;
        a.part = part;
        a.ms = ppl::MSplit{mg.tiles_m, mg.base, mg.rem};
        const int items = mg.tiles_m * ((N + ppl::BN - 1) / ppl::BN) * sc.splitk;
        const int grid = std::min(items, p->num_sms);
        switch (mg.ni) {
#define PPL_LAUNCH_NI(NI)                                                                                   \
    case NI:                                                                                                \
        ppl::k_step1_tma<NI><<<grid, ppl::TMA_THREADS, ppl::Step1Cfg<NI>::SMEM, s>>>(*mapA, *mapB, a);    \
        break;
            PPL_LAUNCH_NI(1) PPL_LAUNCH_NI(2) PPL_LAUNCH_NI(3) PPL_LAUNCH_NI(4) PPL_LAUNCH_NI(5) PPL_LAUNCH_NI(6) PPL_LAUNCH_NI(7)
            PPL_LAUNCH_NI(8) PPL_LAUNCH_NI(9) PPL_LAUNCH_NI(10)
#undef PPL_LAUNCH_NI
            default: return fail(PPL_ERR_INVALID_ARG);
        }
    } else {
        ppl::Step1Args a;
        a.A = A;
        a.B = B;
        a.lda = lda;
        a.ldb = ldb;
        a.M = M;
        a.N = N;
        a.K = (int)K;
        a.k_per_split = sc.k_per_split;
        a.part = part;
        dim3 grid(((M + ppl::BM - 1) / ppl::BM) * ((N + ppl::BN - 1) / ppl::BN), sc.splitk);
        if (vec16)
            ppl::k_step1<2><<<grid, ppl::NTHREADS, ppl::SMEM_K, s>>>(a);
        else
            ppl::k_step1<1><<<grid, ppl::NTHREADS, ppl::SMEM_K, s>>>(a);
    }
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

ppl::RStrides r_strides(int o, int v, int layout) {
    ppl::RStrides s;
    if (layout == PPL_LAYOUT_IAJB) {  // [i][a][j][b]
        s.i = (int64_t)v * o * v;
        s.a = (int64_t)o * v;
        s.j = v;
        s.b = 1;
    } else {  // [i][j][a][b]
        s.i = (int64_t)o * v * v;
        s.j = (int64_t)v * v;
        s.a = v;
        s.b = 1;
    }
    return s;
}

int launch_reduce(const ppl_plan_s *p, const Tile &t, int splitk, int n_rows, int n_off, int tb, double *R,
                  const ppl_opts_t &o, cudaStream_t s) {
    ppl::ReduceArgs a;
    a.part = p->part;
    a.splitk = splitk;
    a.M = p->o * p->o;
    a.N = n_rows;
    a.o = p->o;
    a.v = p->v;
    a.tb = tb;
    a.a0 = t.a0;
    a.b0 = t.b0;
    a.n_off = n_off;
    a.mirror = t.mirror;
    a.alpha = o.alpha;
    a.beta = o.beta;
    a.rs = r_strides(p->o, p->v, o.r_layout);
    a.R = R;
    const int64_t MN = (int64_t)a.M * a.N;
    const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
    ppl::k_reduce<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int launch_reduce_sa(const ppl_plan_s *p, const Tile &t, const double *partp, const double *partm, double *R,
                     const ppl_opts_t &o, cudaStream_t s) {
    ppl::ReduceSaArgs a;
    a.partp = partp;
    a.partm = partm;
    a.sp = t.sp.splitk;
    a.sm = (p->Mm > 0 && p->Km > 0) ? t.sm.splitk : 0;
    a.Mp = p->Mp;
    a.Mm = p->Mm;
    a.N = t.ta * t.tb;
    a.o = p->o;
    a.v = p->v;
    a.tb = t.tb;
    a.a0 = t.a0;
    a.b0 = t.b0;
    a.mirror = t.mirror;
    a.alpha = o.alpha;
    a.beta = o.beta;
    a.rs = r_strides(p->o, p->v, o.r_layout);
    a.R = R;
    const int64_t MN = (int64_t)a.Mp * a.N;
    const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
    ppl::k_reduce_sa<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// W tile X [rows][vv] -> W+ [rows][ldp], W- [rows][ldm]
int launch_fold(const ppl_plan_s *p, const double *X, int rows, double *Wp, double *Wm, cudaStream_t s) {
    ppl::FoldArgs a;
    a.src = X;
    a.sc = p->v;
    a.s_row = p->vv;
    a.s_i = a.s_j = 0;
    a.mode = 0;
    a.rows = rows;
    a.row0 = 0;
    a.o = p->o;
    a.v = p->vp;
    a.vs = p->v;
    a.scale = 1.0;
    a.diag = 1.0;
    a.tbp = a.bg0 = a.A0 = a.ta = 0;
    a.cb_min = 0;
    a.dp = Wp;
    a.dm = Wm;
    a.ldp = p->ldp;
    a.ldm = p->ldm;
    const int nbv = (p->vp + ppl::FT - 1) / ppl::FT;
    dim3 grid(nbv * (nbv + 1) / 2, ppl::fold_grid_y(nbv * (nbv + 1) / 2, rows, p->num_sms));
    ppl::k_symfold<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// t2 (either storage order) -> tau+ [Mp][ldp], tau- [Mm][ldm]
// rows [row0, row1) of the flattened (i,j) index (default: all).  t2 is the address of element (0,0,0,0) and roff_bias 0; when
// the amplitudes are packed chunk by chunk (ppl_apply_host) t2 is the staged chunk's own base and roff_bias the number of
// elements the array would have in front of it (row0 * nvirt^2): no pointer outside the chunk is ever formed
int launch_pack(const ppl_plan_s *p, const double *t2, int layout, double diag, cudaStream_t s, int row0 = 0, int row1 = -1,
                int64_t roff_bias = 0) {
    ppl::FoldArgs a;
    a.src = t2;
    a.roff_bias = roff_bias;
    const ppl::RStrides ts = r_strides(p->o, p->v, layout);  // t2[i,j,c,d] has the strides of R[i,j,a,b]
    a.sc = ts.a;
    a.s_row = 0;
    a.s_i = ts.i;
    a.s_j = ts.j;
    a.mode = 1;
    a.rows = row1 >= 0 ? row1 : p->o * p->o;
    a.row0 = row0;
    a.o = p->o;
    a.v = p->vp;
    a.vs = p->v;
    a.scale = 0.5;
    a.diag = diag;
    a.tbp = a.bg0 = a.A0 = a.ta = 0;
    a.cb_min = 0;
    a.dp = p->taup;
    a.dm = p->taum;
    a.ldp = p->ldp;
    a.ldm = p->ldm;
    const int nbv = (p->vp + ppl::FT - 1) / ppl::FT;
    dim3 grid(nbv * (nbv + 1) / 2, ppl::fold_grid_y(nbv * (nbv + 1) / 2, a.rows - a.row0, p->num_sms));
    ppl::k_symfold<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// The plan's workspace, streams and events belong to the device ppl_plan ran on; a call from a thread whose current device
// is another one would launch there against this device's memory.
bool device_ok(const ppl_plan_s *p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return dev == p->device;
}

int check_ptrs(const ppl_plan_s *p, const double *L, const double *t2, const double *R, bool *vec16) {
    if (!p || !L || !t2 || !R) return PPL_ERR_INVALID_ARG;
    if (!device_ok(p)) return PPL_ERR_INVALID_ARG;
    const uintptr_t all = (uintptr_t)L | (uintptr_t)t2 | (uintptr_t)R;
    if (all & 7) return PPL_ERR_INVALID_ARG;
    *vec16 = p->vec16 && ((all & 15) == 0);
    return PPL_OK;
}

int check_opts(const ppl_opts_t *in, ppl_opts_t *out) {
    out->t2_layout = PPL_LAYOUT_IJAB;
    out->r_layout = PPL_LAYOUT_IJAB;
    out->alpha = 1.0;
    out->beta = 1.0;
    if (!in) return PPL_OK;
    if ((in->t2_layout != PPL_LAYOUT_IJAB && in->t2_layout != PPL_LAYOUT_IAJB) ||
        (in->r_layout != PPL_LAYOUT_IJAB && in->r_layout != PPL_LAYOUT_IAJB))
        return PPL_ERR_INVALID_ARG;
    *out = *in;
    return PPL_OK;
}

// un-packed modes: t2 as the [(i,j)][(c,d)] matrix step 1 reads; a 'iajb'-stored t2 is permuted into tperm
int t2_matrix(ppl_plan_s *p, const double *t2, int layout, cudaStream_t s, const double **out) {
    *out = t2;
    if (layout == PPL_LAYOUT_IJAB) return PPL_OK;
    const size_t bytes = (size_t)p->o * p->o * p->vv * 8;
    if (!p->tperm && cudaMalloc(&p->tperm, bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        p->tperm = nullptr;
        return fail(PPL_ERR_ALLOC);
    }
    ppl::k_permute_t2<<<p->num_sms * 8, 256, 0, s>>>(t2, p->tperm, p->o, p->v);
    PPL_CUDA(cudaGetLastError());
    *out = p->tperm;
    return PPL_OK;
}

// per-launch event log of ppl_apply_profiled
enum Kind { K_PACK = 0, K_STEP0, K_FOLD, K_STEP1, K_REDUCE, K_KINDS };
struct Prof {
    std::vector<cudaEvent_t> ev;
    std::vector<int> kind;
    int launches[K_KINDS] = {0, 0, 0, 0, 0};
    int mark(int k, int n_launches, cudaStream_t s) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return PPL_ERR_CUDA;
        ev.push_back(e);
        kind.push_back(k);
        if (k >= 0) launches[k] += n_launches;
        return cudaEventRecord(e, s) == cudaSuccess ? PPL_OK : PPL_ERR_CUDA;
    }
};

// The whole path.  prof == nullptr: two streams, W-tile ring (the product path).  prof != nullptr: one
// stream, one slot, an event after every stage (measurement only).
int run_apply(ppl_plan_s *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts_in, cudaStream_t stream,
              Prof *prof) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, t2, R, &vec16);
    ppl_opts_t opts;
    if (rc == PPL_OK) rc = check_opts(opts_in, &opts);
    if (rc != PPL_OK) return fail(rc);
    const int ntiles = (int)p->tiles.size();
    const bool sa = p->sym == PPL_SYM_PAIR_SA;
    const bool tma0 = p->use_tma && vec16;             // step 0 reads the caller's L: needs 16-byte rows
    const bool tma1 = sa ? p->use_tma != 0 : tma0;     // SA step 1 reads plan-owned, padded operands
    const bool two_streams = !prof && p->ring >= 2 && ntiles >= 2;
    cudaStream_t gen = two_streams ? p->gen : stream;
#define PPL_MARK(k, n)                                                         \
    do {                                                                       \
        if (prof && prof->mark(k, n, stream) != PPL_OK) return fail(PPL_ERR_CUDA); \
    } while (0)

    if (two_streams) {  // fork: the producer stream starts after prior work on `stream`
        PPL_CUDA(cudaEventRecord(p->ev_in, stream));
        PPL_CUDA(cudaStreamWaitEvent(gen, p->ev_in, 0));
    }
    PPL_MARK(-1, 0);
    const double *t2m = t2;
    if (sa) {
        if ((rc = launch_pack(p, t2, opts.t2_layout, 1.0, stream)) != PPL_OK) return rc;
        PPL_MARK(K_PACK, 1);
    } else if (opts.t2_layout != PPL_LAYOUT_IJAB) {
        if ((rc = t2_matrix(p, t2, opts.t2_layout, stream, &t2m)) != PPL_OK) return rc;
        PPL_MARK(K_PACK, 1);
    }
    CUtensorMap mapL, mapT;
    if (tma0 && make_map_2d(&mapL, L, (uint64_t)p->vv, (uint64_t)p->x, (uint64_t)p->vv * 8, 16, ppl::BK) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    if (!sa && tma1 &&
        make_map_2d(&mapT, t2m, (uint64_t)p->vv, (uint64_t)p->o * p->o, (uint64_t)p->vv * 8, ppl::BK, (uint32_t)p->bm_full) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    const bool minus = sa && p->Mm > 0 && p->Km > 0;

    for (int k = 0; k < ntiles; ++k) {
        const Tile &t = p->tiles[k];
        const int slot = prof ? 0 : k % p->ring;
        const int N = t.ta * t.tb;
        double *Wp = p->slot[slot], *Wm = p->slot[slot] + (size_t)p->T * p->T * p->ldp;
        if (two_streams && k >= p->ring) PPL_CUDA(cudaStreamWaitEvent(gen, p->ev_free[slot], 0));
        // ---- producer: step 0 (and the +- fold) ----
        if ((rc = launch_step0(p, t, L, tma0 ? &mapL : nullptr, sa ? p->X : p->slot[slot], vec16, gen)) != PPL_OK) return rc;
        PPL_MARK(K_STEP0, 1);
        if (sa) {
            if ((rc = launch_fold(p, p->X, N, Wp, Wm, gen)) != PPL_OK) return rc;
            PPL_MARK(K_FOLD, 1);
        }
        if (two_streams) {
            PPL_CUDA(cudaEventRecord(p->ev_ready[slot], gen));
            PPL_CUDA(cudaStreamWaitEvent(stream, p->ev_ready[slot], 0));
        }
        // ---- consumer: step 1, reduce ----
        if (sa) {
            double *partp = p->part, *partm = p->part + (size_t)t.sp.splitk * p->Mp * N;
            rc = launch_step1(p, tma1 ? &p->mapTp : nullptr, tma1 ? &p->mapWp[slot] : nullptr, p->mg_p, p->taup, p->ldp, Wp,
                              p->ldp, p->Mp, N, p->Kp, t.sp, partp, true, stream);
            if (rc == PPL_OK && minus)
                rc = launch_step1(p, tma1 ? &p->mapTm : nullptr, tma1 ? &p->mapWm[slot] : nullptr, p->mg_m, p->taum, p->ldm,
                                  Wm, p->ldm, p->Mm, N, p->Km, t.sm, partm, true, stream);
            if (rc != PPL_OK) return rc;
            PPL_MARK(K_STEP1, minus ? 2 : 1);
            if (two_streams) PPL_CUDA(cudaEventRecord(p->ev_free[slot], stream));
            if ((rc = launch_reduce_sa(p, t, partp, partm, R, opts, stream)) != PPL_OK) return rc;
        } else {
            rc = launch_step1(p, tma1 ? &mapT : nullptr, tma1 ? &p->mapW[slot] : nullptr, p->mg_full, t2m, p->vv, p->slot[slot],
                              p->vv, p->o * p->o, N, p->vv, t.full, p->part, vec16, stream);
            if (rc != PPL_OK) return rc;
            PPL_MARK(K_STEP1, 1);
            if (two_streams) PPL_CUDA(cudaEventRecord(p->ev_free[slot], stream));
            if ((rc = launch_reduce(p, t, t.full.splitk, N, 0, t.tb, R, opts, stream)) != PPL_OK) return rc;
        }
        PPL_MARK(K_REDUCE, 1);
    }
#undef PPL_MARK
    // join: every producer launch is followed by a consumer wait on `stream`, so `stream` already
    // depends on all work of `gen`.
    return PPL_OK;
}


// ------------------------------------------------------------------------------------------
// PPL_SYM_FULL (ppl_kernels_full.cuh): slabs of 16 a's, tiles (A; b-group), chunk table of step 0.
// ------------------------------------------------------------------------------------------
// Allocate what full_plan sized (device half).  Sets full_ok, or leaves it 0 (the plan then stays without PPL_SYM_FULL).
int full_allocate(ppl_plan_s *p) {
    p->full_ok = 0;
    if (!p->full_planned) return PPL_OK;
    const int TA = ppl::TA_FULL;
    const size_t x_bytes = p->fx_bytes, lq_bytes = p->lq_bytes, lpad_bytes = p->lpad_bytes;
    const bool two_strips = p->two_strips;
    const std::vector<int2> &chunks = p->chunks_host;
    const size_t racc_bytes = p->tau_bytes;
    if (cudaMalloc(&p->fws, p->fws_bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        p->fws = nullptr;
        return PPL_OK;
    }
    if (cudaMemset(p->fws, 0, p->fws_bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        return PPL_OK;
    }
    const size_t slot_rows = (size_t)TA * p->tbg + 16;
    unsigned char *q = p->fws;
    p->fX = reinterpret_cast<double *>(q);
    q += x_bytes;
    for (int s = 0; s < p->fslots; ++s) {
        p->fWp[s] = reinterpret_cast<double *>(q);
        q += align256(slot_rows * p->ldp * 8);
        p->fWm[s] = reinterpret_cast<double *>(q);
        q += align256(slot_rows * p->ldm * 8);
    }
    p->fpart = reinterpret_cast<double *>(q);
    q += align256(p->fpart_bytes);
    p->raccp = reinterpret_cast<double *>(q);
    p->raccm = reinterpret_cast<double *>(q + align256((size_t)p->Mp * p->ldp * 8));
    q += racc_bytes;
    p->fchunks = reinterpret_cast<int2 *>(q);
    q += align256(chunks.size() * sizeof(int2));
    p->Lpad = lpad_bytes ? reinterpret_cast<double *>(q) : nullptr;
    q += lpad_bytes;
    p->Lq = lq_bytes ? reinterpret_cast<double *>(q) : nullptr;
    q += lq_bytes;
    p->fX2 = two_strips ? reinterpret_cast<double *>(q) : nullptr;
    if (cudaMemcpy(p->fchunks, chunks.data(), chunks.size() * sizeof(int2), cudaMemcpyHostToDevice) != cudaSuccess) {
        (void)cudaGetLastError();
        return PPL_OK;
    }
    const uint64_t rows = slot_rows;
    bool m = true;
    for (int s = 0; s < p->fslots; ++s) {
        m = m && make_map_2d(&p->mapFWp[s], p->fWp[s], (uint64_t)p->Kp, rows, (uint64_t)p->ldp * 8, ppl::BK, ppl::BN) == PPL_OK;
        m = m && make_map_2d(&p->mapFWpT[s], p->fWp[s], (uint64_t)p->Kp, rows, (uint64_t)p->ldp * 8, 16, ppl::BK) == PPL_OK;
        if (p->Km > 0) {
            m = m && make_map_2d(&p->mapFWm[s], p->fWm[s], (uint64_t)p->Km, rows, (uint64_t)p->ldm * 8, ppl::BK, ppl::BN) == PPL_OK;
            m = m && make_map_2d(&p->mapFWmT[s], p->fWm[s], (uint64_t)p->Km, rows, (uint64_t)p->ldm * 8, 16, ppl::BK) == PPL_OK;
        }
    }
    if (p->Lq) m = m && make_map_2d(&p->mapLq, p->Lq, (uint64_t)p->ldq, (uint64_t)p->x, (uint64_t)p->ldq * 8, 16, ppl::BK) == PPL_OK;
    if (!m) return PPL_OK;
    bool ok = true;
    for (int i = 0; i < 4 && ok; ++i) ok = ok && cudaStreamCreateWithFlags(&p->fs[i], cudaStreamNonBlocking) == cudaSuccess;
    if (p->fX2) {
        ok = ok && cudaStreamCreateWithFlags(&p->fs0, cudaStreamNonBlocking) == cudaSuccess;  // (stream priorities either way: no gain, measured)
        ok = ok && cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) == cudaSuccess;
        for (int s = 0; s < 2 && ok; ++s) {
            ok = ok && cudaEventCreateWithFlags(&p->ev_s0[s], cudaEventDisableTiming) == cudaSuccess;
            ok = ok && cudaEventCreateWithFlags(&p->ev_xfree[s], cudaEventDisableTiming) == cudaSuccess;
        }
    }
    for (int s = 0; s < 2 && ok; ++s) {
        ok = ok && cudaEventCreateWithFlags(&p->ev_fold[s], cudaEventDisableTiming) == cudaSuccess;
        for (int i = 0; i < 4 && ok; ++i) ok = ok && cudaEventCreateWithFlags(&p->evg[s][i], cudaEventDisableTiming) == cudaSuccess;
    }
    if (!ok) {
        (void)cudaGetLastError();
        return PPL_OK;
    }
    p->full_ok = 1;
    return PPL_OK;
}

int launch_step1t(const ppl_plan_s *p, const CUtensorMap *mapA, const CUtensorMap *mapB, const MGeom &mg, int M, const FullTile &t,
                  bool minus, double *acc, int64_t ld, cudaStream_t s) {
    ppl::Step1TArgs a;
    a.M = M;
    a.n_begin = minus ? t.k1m : t.k1p;
    a.n_end = minus ? p->Km : p->Kp;
    a.n_base = a.n_begin & ~15;
    if (M <= 0 || a.n_end - a.n_begin <= 0) return PPL_OK;
    a.range = t.range;
    a.kap0 = minus ? t.km0 : t.kp0;
    a.kt_per_a = t.range ? 1 : t.tbp / 16;
    a.nkt = t.range ? (minus ? t.nmr : t.npr) / 16 : ppl::TA_FULL * a.kt_per_a;
    if (a.nkt <= 0) return PPL_OK;
    a.A0 = t.A0;
    a.bg0 = t.bg0;
    a.v = p->vp;
    a.minus = minus ? 1 : 0;
    a.acc = acc;
    a.ld = ld;
    a.ms = ppl::MSplit{mg.tiles_m, mg.base, mg.rem};
    const int items = mg.tiles_m * ((a.n_end - a.n_base + ppl::BN - 1) / ppl::BN);
    const int grid = std::min(items, p->num_sms);
    switch (mg.ni) {
#define PPL_LAUNCH_NI(NI)                                                                                  \
    case NI:                                                                                               \
        ppl::k_step1t_tma<NI><<<grid, ppl::TMA_THREADS, ppl::Step1Cfg<NI>::SMEM, s>>>(*mapA, *mapB, a);  \
        break;
        PPL_LAUNCH_NI(1) PPL_LAUNCH_NI(2) PPL_LAUNCH_NI(3) PPL_LAUNCH_NI(4) PPL_LAUNCH_NI(5) PPL_LAUNCH_NI(6) PPL_LAUNCH_NI(7)
            PPL_LAUNCH_NI(8) PPL_LAUNCH_NI(9) PPL_LAUNCH_NI(10)
#undef PPL_LAUNCH_NI
        default: return fail(PPL_ERR_INVALID_ARG);
    }
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int launch_reduce_acc(const ppl_plan_s *p, const FullTile &t, const double *part, int splitk, int M, bool minus, double *acc,
                      int64_t ld, cudaStream_t s) {
    if (M <= 0 || splitk <= 0) return PPL_OK;
    if (t.range) {
        ppl::ReduceRangeArgs a;
        a.part = part;
        a.splitk = splitk;
        a.M = M;
        a.N = minus ? t.nm : t.np;
        a.k0 = minus ? t.km0 : t.kp0;
        a.acc = acc;
        a.ld = ld;
        if (a.N <= 0) return PPL_OK;
        const int64_t MN = (int64_t)a.M * a.N;
        const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
        ppl::k_reduce_range<<<grid, 256, 0, s>>>(a);
        PPL_CUDA(cudaGetLastError());
        return PPL_OK;
    }
    ppl::ReduceAccArgs a;
    a.part = part;
    a.splitk = splitk;
    a.M = M;
    a.N = ppl::TA_FULL * t.tbp;
    a.tbp = t.tbp;
    a.A0 = t.A0;
    a.ta = t.ta;
    a.bg0 = t.bg0;
    a.v = p->vp;
    a.minus = minus ? 1 : 0;
    a.acc = acc;
    a.ld = ld;
    const int64_t MN = (int64_t)a.M * a.N;
    const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
    ppl::k_reduce_acc<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// L2 policy bits of step 0 (ppl_debug_opts_t.full_hints: 0 = the default 1 + 4 + 8, -1 = none)
inline int step0_hints(const ppl_plan_s *p) { return p->dbg.full_hints == 0 ? 13 : (p->dbg.full_hints < 0 ? 0 : p->dbg.full_hints); }

// The whole path in PPL_SYM_FULL: everything on the caller's stream (every kernel fills the GPU; the
// strip is single-buffered), prof as in run_apply.
enum { FULL_PACK = 1, FULL_COMPUTE = 2, FULL_UNPACK = 4, FULL_ALL = 7 };
int launch_unpack_full(const ppl_plan_s *p, const ppl_opts_t &opts, double *R, int64_t idx0, int64_t idx1, cudaStream_t stream,
                       int a0 = 0, int na = -1, const ppl::RStrides *rs = nullptr, int64_t r_bias = 0);

// phases: FULL_PACK (t2 -> tau+-, clear R+-acc), FULL_COMPUTE (all slabs), FULL_UNPACK (R+-acc -> R).  ppl_apply runs all
// three; ppl_apply_host packs and unpacks chunk by chunk itself and calls this with FULL_COMPUTE only (t2, R unused).
// tau_ready (ppl_apply_host): tau+- are being packed on other streams; step 0 of the first slab needs only L and starts at
// once, the event is waited for behind it.
int run_apply_full(ppl_plan_s *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts_in, cudaStream_t stream,
                   Prof *prof, int phases = FULL_ALL, cudaEvent_t tau_ready = nullptr, const pplapi::SlabHook *hook = nullptr) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, (phases & FULL_PACK) ? t2 : L, (phases & FULL_UNPACK) ? R : L, &vec16);
    ppl_opts_t opts;
    if (rc == PPL_OK) rc = check_opts(opts_in, &opts);
    // only L is read by TMA (16-byte aligned rows, or the padded copy); t2 and R are packed / unpacked with scalar accesses
    if (rc == PPL_OK && (!p->full_ok || (((uintptr_t)L & 15) != 0 && !p->Lpad))) rc = PPL_ERR_INVALID_ARG;
    if (rc != PPL_OK) return fail(rc);
#define PPL_MARK(k, n)                                                             \
    do {                                                                           \
        if (prof && prof->mark(k, n, stream) != PPL_OK) return fail(PPL_ERR_CUDA); \
    } while (0)
    PPL_MARK(-1, 0);
    const bool dbg = p->dbg.debug_sync != 0;  // debug: synchronise and report after every launch
#define PPL_DBG(label, k)                                                                              \
    do {                                                                                               \
        if (dbg) {                                                                                     \
            const cudaError_t e__ = cudaStreamSynchronize(stream);                                     \
            if (e__ != cudaSuccess) {                                                                  \
                fprintf(stderr, "libppl: %s (tile/slab %d) failed: %s\n", label, (int)(k), cudaGetErrorString(e__)); \
                return fail(PPL_ERR_CUDA);                                                             \
            }                                                                                          \
        }                                                                                              \
    } while (0)
    const bool minus = p->Mm > 0 && p->Km > 0;
    if (phases & FULL_PACK) {
        if ((rc = launch_pack(p, t2, opts.t2_layout, 0.5, stream)) != PPL_OK) return rc;
        PPL_CUDA(cudaMemsetAsync(p->raccp, 0, (size_t)p->Mp * p->ldp * 8, stream));
        if (minus) PPL_CUDA(cudaMemsetAsync(p->raccm, 0, (size_t)p->Mm * p->ldm * 8, stream));
        PPL_MARK(K_PACK, 1);
    }
    if (!(phases & FULL_COMPUTE)) return PPL_OK;
    if (p->Lpad) {  // odd nvirt: L -> [x][vp][vp] with a zero pad row / column (2 x |L| bytes of HBM traffic, << 1 % of an apply)
        ppl::k_pad_L<<<p->num_sms * 8, 256, 0, stream>>>(L, p->Lpad, p->x, p->v, p->vp);
        PPL_CUDA(cudaGetLastError());
        PPL_MARK(K_PACK, 1);
        L = p->Lpad;
    }
    CUtensorMap mapL;
    if (make_map_2d(&mapL, L, (uint64_t)p->vvp, (uint64_t)p->x, (uint64_t)p->vvp * 8, 16, ppl::BK, (step0_hints(p) & 8) != 0) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    if (p->Lq && p->diag_pack && !p->full_tight) {  // the diagonal 16 x 16 blocks of L, pairs b <= d only (|L| / (nvirt / 16) bytes)
        const int64_t total = (int64_t)p->x * p->nfull * ppl::DIAG_PACKED;
        const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)p->num_sms * 8);
        ppl::k_pack_diag<<<std::max(grid, 1), 256, 0, stream>>>(L, p->Lq, p->x, p->vp, p->nfull, p->ldq);
        PPL_CUDA(cudaGetLastError());
        PPL_MARK(K_PACK, 1);
    }
    const int TA = ppl::TA_FULL;
    const bool serial = p->dbg.full_serial != 0;  // debug: everything on the caller's stream
    const bool conc = !prof && !dbg && !serial;
    // PPL_TRACE (debug): a timed event pair around every launch ON ITS OWN STREAM -- the concurrency is kept -- and a
    // timeline on stderr after a synchronise: "label index stream t_eligible_ms t_end_ms" (t_eligible: the stream has
    // reached the launch, i.e. its predecessors and awaited events are complete).
    static const bool trace_env = getenv("PPL_TRACE") != nullptr;
    const bool trace = (trace_env || p->dbg.trace) && conc;
    struct TraceRec {
        const char *label;
        int k, sid;
        cudaEvent_t b, e;
    };
    std::vector<TraceRec> tr;
    auto tb = [&](const char *label, int k, int sid, cudaStream_t st) {
        if (!trace) return;
        TraceRec r{label, k, sid, nullptr, nullptr};
        cudaEventCreate(&r.b);
        cudaEventCreate(&r.e);
        cudaEventRecord(r.b, st);
        tr.push_back(r);
    };
    auto te = [&](cudaStream_t st) {
        if (trace) cudaEventRecord(tr.back().e, st);
    };
    int tile_no = 0;
    // Two strips: step 0 runs on its own stream, one slab ahead of the folds (strip k & 1), so that the HBM-bound fold of
    // slab k and the tail of its GEMMs are filled by the DMMA work of slab k + 1 instead of standing between two slabs.
    const bool dual = conc && p->fX2 != nullptr;
    cudaStream_t s0 = dual ? p->fs0 : stream;
    if (dual) {  // fork: step 0 starts behind everything queued on `stream` so far (the padded copy of L included)
        PPL_CUDA(cudaEventRecord(p->ev_fork, stream));
        PPL_CUDA(cudaStreamWaitEvent(s0, p->ev_fork, 0));
    }
    // One unit of step 0: a slab (the whole strip: d-block >= b-block plus the b<->d image) or, in the memory-tight mode,
    // one (slab; b-group) tile on its full (b, d) rectangle.  Unit u writes strip u & 1 when there are two.
    const bool tight = p->full_tight != 0;
    int unit_no = 0, xi = 0;
    double *X = p->fX;
    auto step0_unit = [&](const FullSlab &sl, const FullTile *t) -> int {
        xi = dual ? (unit_no & 1) : 0;
        X = xi ? p->fX2 : p->fX;
        ppl::Step0SlabArgs a0;
        a0.A0 = sl.A0;
        a0.ta = sl.ta;
        a0.v = p->vp;
        a0.K = p->x;
        a0.tiles_m = sl.tiles_m;
        a0.tiles_n = t ? t->tiles_n : sl.tiles_n;
        a0.chunks = p->fchunks + (t ? t->chunk_off : sl.chunk_off);
        a0.X = X;
        a0.rows_per_a = t ? t->tbp : p->vp;
        a0.b_base = t ? t->bg0 : 0;
        a0.image = t ? 0 : 1;
        // Raster and L2 policy of step 0, from ncu's DRAM bytes of one slab (profiles/r02_step0_l2.md): the 148 persistent CTAs
        // drift apart, so a panel is shared only while it survives in L2.  Groups of 12 row tiles (a wave covers ~12 x 12 tiles:
        // the fewest panels per wave), 128-byte instead of 256-byte L2 promotion of the TMA loads (a box row is 128 bytes: the
        // promoted other half belongs to a column tile that runs much later), evict_last on the row panels and streaming
        // stores of the strip: 204 -> 82 GB read per slab at XL, 7.5 -> 3.5 GB at large, same kernel time (DMMA-bound).
        a0.group_m = p->dbg.full_group_m > 0 ? p->dbg.full_group_m : ppl::GROUP_M;
        a0.hints = step0_hints(p) & 7;
        const int items = a0.tiles_m * a0.tiles_n;
        if (dual && unit_no >= 2) PPL_CUDA(cudaStreamWaitEvent(s0, p->ev_xfree[xi], 0));  // the folds of unit u - 2 have read this strip
        tb("step0", t ? t->bg0 : sl.A0, 0, s0);
        ppl::k_step0_slab<<<std::min(items, p->num_sms), ppl::TMA_THREADS, ppl::SMEM_TMA, s0>>>(mapL, p->Lq ? p->mapLq : mapL, a0);
        te(s0);
        PPL_CUDA(cudaGetLastError());
        PPL_DBG("k_step0_slab", sl.A0);
        PPL_MARK(K_STEP0, 1);
        if (dual) {
            PPL_CUDA(cudaEventRecord(p->ev_s0[xi], s0));
            PPL_CUDA(cudaStreamWaitEvent(stream, p->ev_s0[xi], 0));
        }
        if (tau_ready && unit_no == 0) PPL_CUDA(cudaStreamWaitEvent(stream, tau_ready, 0));
        return PPL_OK;
    };
    auto unit_done = [&]() -> int {  // behind the last fold that reads the unit's strip
        if (dual) PPL_CUDA(cudaEventRecord(p->ev_xfree[xi], stream));
        ++unit_no;
        return PPL_OK;
    };
    for (const FullSlab &sl : p->slabs) {
        if (!tight && (rc = step0_unit(sl, nullptr)) != PPL_OK) return rc;
        for (int k = sl.tile_begin; k < sl.tile_end; ++k) {
            const FullTile &t = p->ftiles[k];
            const int N = t.range ? t.np : TA * t.tbp;   // W+ rows contracted by use 1
            const int Nm = t.range ? t.nm : TA * t.tbp;  // W- rows
            if (tight && (rc = step0_unit(sl, &t)) != PPL_OK) return rc;
            const int sl_w = conc ? (tile_no % p->fslots) : 0;  // W+- slot of this tile
            if (conc && tile_no >= p->fslots)  // the GEMMs of the tile that used this slot last still read it
                for (int i = 0; i < 4; ++i) PPL_CUDA(cudaStreamWaitEvent(stream, p->evg[sl_w][i], 0));
            {   // fold: strip rows -> W+- tile
                ppl::FoldArgs f;
                f.src = X;
                f.sc = p->vp;
                f.s_row = p->vvp;
                f.s_i = f.s_j = 0;
                f.mode = t.range ? 3 : 2;
                f.rows = t.range ? t.npr + t.nzm : N;
                f.row0 = 0;
                f.kp0 = t.kp0;
                f.kp1 = t.kp0 + t.np;
                f.km0 = t.km0;
                f.nzm = t.nzm;
                for (int z = 0; z < t.nzm; ++z) f.zrows_m[z] = t.zrows_m[z];
                f.o = p->o;
                f.v = f.vs = p->vp;
                f.scale = 1.0;
                f.diag = 2.0;
                f.tbp = t.tbp;
                f.rows_per_a = tight ? t.tbp : p->vp;
                f.b_base = tight ? t.bg0 : 0;
                f.bg0 = t.bg0;
                f.A0 = t.A0;
                f.ta = t.ta;
                f.cb_min = t.A0 / ppl::FT;
                f.dp = p->fWp[sl_w];
                f.dm = p->fWm[sl_w];
                f.ldp = p->ldp;
                f.ldm = p->ldm;
                const int nb = (p->vp + ppl::FT - 1) / ppl::FT - f.cb_min;
                dim3 grid(nb * (nb + 1) / 2, ppl::fold_grid_y(nb * (nb + 1) / 2, f.rows, p->num_sms));
                tb("fold", k, 1, stream);
                ppl::k_symfold<<<grid, 256, 0, stream>>>(f);
                te(stream);
                PPL_CUDA(cudaGetLastError());
                PPL_DBG("k_symfold", k);
                PPL_MARK(K_FOLD, 1);
                if (tight && (rc = unit_done()) != PPL_OK) return rc;
            }
            // The four GEMMs of the tile are independent given the fold (use 1 writes the R+-acc columns of the slab,
            // use 2 those above it; + and - are different matrices): outside the profiled pass each runs on a side
            // stream of its own, so that the tail of one persistent kernel is filled by the CTAs of the next, and the
            // next slab's step 0 (ordered only behind this slab's last fold: it overwrites the strip) fills theirs.
            cudaStream_t g0 = conc ? p->fs[0] : stream, g1 = conc ? p->fs[1] : stream, g2 = conc ? p->fs[2] : stream,
                         g3 = conc ? p->fs[3] : stream;
            if (conc) {
                PPL_CUDA(cudaEventRecord(p->ev_fold[sl_w], stream));
                for (int i = 0; i < 4; ++i) PPL_CUDA(cudaStreamWaitEvent(p->fs[i], p->ev_fold[sl_w], 0));
            }
            // use 1: R+-acc[.][(a,b)] += tau+-[.][J >= (A0,A0)] W+-[(a,b)][J]^T
            double *partp = p->fpart, *partm = p->fpart + p->fpart_m_off;
            tb("use1+", k, 2, g0);
            rc = launch_step1(p, &p->mapTp, &p->mapFWp[sl_w], p->mg_p, nullptr, 0, nullptr, 0, p->Mp, N, p->Kp, t.sp, partp, true, g0,
                              t.k0p);
            te(g0);
            const bool m1 = minus && p->Km - t.k0m > 0 && Nm > 0;
            if (rc == PPL_OK && m1) {
                tb("use1-", k, 3, g1);
                rc = launch_step1(p, &p->mapTm, &p->mapFWm[sl_w], p->mg_m, nullptr, 0, nullptr, 0, p->Mm, Nm, p->Km, t.sm, partm, true,
                                  g1, t.k0m);
                te(g1);
            }
            if (rc != PPL_OK) return rc;
            PPL_DBG("use 1 (k_step1_tma)", k);
            PPL_MARK(K_STEP1, m1 ? 2 : 1);
            if (conc && tile_no >= 1) {
                // use 2 of the previous tile (previous slab) adds into the R+-acc columns this reduction updates:
                // order them (with two W+- slots the fold no longer separates consecutive tiles)
                const int prev = (tile_no - 1) % p->fslots;
                PPL_CUDA(cudaStreamWaitEvent(g0, p->evg[prev][2], 0));
                PPL_CUDA(cudaStreamWaitEvent(g1, p->evg[prev][3], 0));
            }
            tb("red+", k, 2, g0);
            rc = launch_reduce_acc(p, t, partp, t.sp.splitk, p->Mp, false, p->raccp, p->ldp, g0);
            te(g0);
            if (rc == PPL_OK && m1) {
                tb("red-", k, 3, g1);
                rc = launch_reduce_acc(p, t, partm, t.sm.splitk, p->Mm, true, p->raccm, p->ldm, g1);
                te(g1);
            }
            if (rc != PPL_OK) return rc;
            PPL_DBG("k_reduce_acc", k);
            PPL_MARK(K_REDUCE, m1 ? 2 : 1);
            // use 2: R+-acc[.][J >= (A0+16,A0+16)] += tau+-[.][(a,b) in tile] W+-[(a,b)][J]
            int n2 = 0;
            if (p->Kp - t.k1p > 0) {
                tb("use2+", k, 4, g2);
                if ((rc = launch_step1t(p, &p->mapTp, &p->mapFWpT[sl_w], p->mg_p, p->Mp, t, false, p->raccp, p->ldp, g2)) != PPL_OK) return rc;
                te(g2);
                PPL_DBG("use 2 plus (k_step1t_tma)", k);
                ++n2;
            }
            if (minus && p->Km - t.k1m > 0 && Nm > 0) {
                tb("use2-", k, 5, g3);
                if ((rc = launch_step1t(p, &p->mapTm, &p->mapFWmT[sl_w], p->mg_m, p->Mm, t, true, p->raccm, p->ldm, g3)) != PPL_OK) return rc;
                te(g3);
                PPL_DBG("use 2 minus (k_step1t_tma)", k);
                ++n2;
            }
            if (n2) PPL_MARK(K_STEP1, n2);
            if (conc)
                for (int i = 0; i < 4; ++i) PPL_CUDA(cudaEventRecord(p->evg[sl_w][i], p->fs[i]));
            ++tile_no;
        }
        if (!tight && (rc = unit_done()) != PPL_OK) return rc;
        // the R+-acc columns (a, b >= a) of this slab's a's are final once its last reductions have run: they were the last
        // writers (use 2 of every earlier slab is ordered before them), later slabs add to later columns only
        if (hook && (rc = hook->fn(hook->ctx, sl.A0, sl.ta, conc ? p->fs[0] : stream, conc ? p->fs[1] : stream)) != PPL_OK) return rc;
    }
    if (conc)  // join: the side streams run in order, so the events of the last min(tiles, slots) tiles cover all work
        for (int s = 0; s < std::min(tile_no, p->fslots); ++s)
            for (int i = 0; i < 4; ++i) PPL_CUDA(cudaStreamWaitEvent(stream, p->evg[s][i], 0));
    if (phases & FULL_UNPACK) {
        tb("unpack", 0, 1, stream);
        if ((rc = launch_unpack_full(p, opts, R, 0, (int64_t)p->o * p->o * p->vv, stream)) != PPL_OK) return rc;
        te(stream);
        PPL_DBG("k_unpack_full", 0);
        PPL_MARK(K_REDUCE, 1);
    }
    if (trace && !tr.empty()) {
        if (cudaStreamSynchronize(stream) == cudaSuccess)
            for (const TraceRec &r : tr) {
                float tb_ms = 0, te_ms = 0;
                cudaEventElapsedTime(&tb_ms, tr.front().b, r.b);
                cudaEventElapsedTime(&te_ms, tr.front().b, r.e);
                fprintf(stderr, "PPL_TRACE %-6s %4d s%d %10.4f %10.4f\n", r.label, r.k, r.sid, tb_ms, te_ms);
            }
        for (const TraceRec &r : tr) {
            cudaEventDestroy(r.b);
            cudaEventDestroy(r.e);
        }
    }
#undef PPL_MARK
#undef PPL_DBG
    return PPL_OK;
}

// R[idx] = beta R + alpha (R+ +- R-) for the flattened (i,j,a,b) indices [idx0, idx1); R is the address of element (0,0,0,0)
// na < 0: all a's, R in the caller's layout; else the a's [a0, a0 + na) with R addressed through *rs (a slab buffer: R is its
// own base, r_bias = a0 * rs->a the elements the full array would have in front of it)
int launch_unpack_full(const ppl_plan_s *p, const ppl_opts_t &opts, double *R, int64_t idx0, int64_t idx1, cudaStream_t stream, int a0,
                       int na, const ppl::RStrides *rs, int64_t r_bias) {
    ppl::UnpackArgs u;
    u.rp = p->raccp;
    u.rm = p->raccm;
    u.ldp = p->ldp;
    u.ldm = p->ldm;
    u.o = p->o;
    u.v = p->v;
    u.vk = p->vp;
    u.alpha = opts.alpha;
    u.beta = opts.beta;
    u.rs = rs ? *rs : r_strides(p->o, p->v, opts.r_layout);
    u.R = R;
    u.r_bias = r_bias;
    u.idx0 = idx0;
    u.idx1 = idx1;
    u.a0 = na < 0 ? 0 : a0;
    u.na = na < 0 ? p->v : na;
    const int64_t blocks = (idx1 - idx0 + 255) / 256;
    ppl::k_unpack_full<<<(int)std::min<int64_t>(std::max<int64_t>(blocks, 1), (int64_t)p->num_sms * 8), 256, 0, stream>>>(u);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

ppl_plan_t *ppl_plan(int nocc, int nvirt, int nchol, size_t workspace_bytes) {
    return ppl_plan_ex(nocc, nvirt, nchol, workspace_bytes, nullptr);
}

ppl_plan_t *ppl_plan_ex(int nocc, int nvirt, int nchol, size_t workspace_bytes, const ppl_debug_opts_t *dbg) {
    if (!dims_ok(nocc, nvirt, nchol)) {
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
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) {
        (void)cudaGetLastError();
        fail(PPL_ERR_CUDA);
        return nullptr;
    }
    const size_t auto_cap = (size_t)(0.9 * (double)free_b);
    const size_t cap = workspace_bytes ? std::min(workspace_bytes, auto_cap) : auto_cap;
    const bool use_tma = !(dbg && dbg->cpasync_kernels) && get_encode() != nullptr;
    int rc_host = PPL_OK;
    ppl_plan_s *p = plan_host(nocc, nvirt, nchol, workspace_bytes, cap, prop.multiProcessorCount, use_tma, dbg, &rc_host);
    if (p) p->device = dev;
    if (!p) {
        fail(rc_host);
        return nullptr;
    }
    if (cudaMalloc(&p->ws, p->ws_bytes) != cudaSuccess ||
        cudaHostAlloc(&p->vflags_host, 32 * sizeof(int), cudaHostAllocMapped) != cudaSuccess ||
        cudaMalloc(&p->vdone_dev, 2 * sizeof(int)) != cudaSuccess || cudaMemset(p->vdone_dev, 0, 2 * sizeof(int)) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_verify, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_vq[0], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_vq[1], cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        free_plan(p);
        fail(PPL_ERR_ALLOC);
        return nullptr;
    }
    if (cudaMemset(p->ws, 0, p->ws_bytes) != cudaSuccess) {  // the holes of the packed layouts stay zero for good
        (void)cudaGetLastError();
        free_plan(p);
        fail(PPL_ERR_CUDA);
        return nullptr;
    }
    {
        unsigned char *q = p->ws;
        p->X = reinterpret_cast<double *>(q);
        q += p->x_bytes;
        for (int i = 0; i < p->ring; ++i, q += p->slot_bytes) p->slot[i] = reinterpret_cast<double *>(q);
        p->part = reinterpret_cast<double *>(q);
        q += p->part_bytes;
        if (p->sa_ok) {
            p->taup = reinterpret_cast<double *>(q);
            p->taum = reinterpret_cast<double *>(q + align256((size_t)p->Mp * p->ldp * 8));
        }
    }

    bool ok = cudaStreamCreateWithFlags(&p->gen, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&p->host_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&p->ev_in, cudaEventDisableTiming) == cudaSuccess;
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
        const uint64_t TT = (uint64_t)p->T * p->T;
        bool m = true;
        for (int i = 0; i < p->ring && m; ++i) {
            if (p->vec16) m = m && make_map_2d(&p->mapW[i], p->slot[i], (uint64_t)p->vv, TT, (uint64_t)p->vv * 8, ppl::BK, ppl::BN) == PPL_OK;
            if (p->sa_ok) {
                m = m && make_map_2d(&p->mapWp[i], p->slot[i], (uint64_t)p->Kp, TT, (uint64_t)p->ldp * 8, ppl::BK, ppl::BN) == PPL_OK;
                if (p->Km > 0)
                    m = m && make_map_2d(&p->mapWm[i], p->slot[i] + TT * p->ldp, (uint64_t)p->Km, TT, (uint64_t)p->ldm * 8, ppl::BK,
                                         ppl::BN) == PPL_OK;
            }
        }
        if (p->sa_ok && m) {
            m = m && make_map_2d(&p->mapTp, p->taup, (uint64_t)p->Kp, (uint64_t)p->Mp, (uint64_t)p->ldp * 8, ppl::BK, (uint32_t)p->bm_p) == PPL_OK;
            if (p->Km > 0 && p->Mm > 0)
                m = m && make_map_2d(&p->mapTm, p->taum, (uint64_t)p->Km, (uint64_t)p->Mm, (uint64_t)p->ldm * 8, ppl::BK,
                                     (uint32_t)p->bm_m) == PPL_OK;
        }
        if (!m) {
            (void)cudaGetLastError();
            free_plan(p);
            fail(PPL_ERR_CUDA);
            return nullptr;
        }
    }
    p->sym = p->sa_ok ? PPL_SYM_PAIR_SA : PPL_SYM_PAIR;
    const int rc = build_tiles(p);
    if (rc != PPL_OK) {
        free_plan(p);
        fail(rc);
        return nullptr;
    }
    // PPL_SYM_FULL: its buffers are allocated when they fit under the cap; it is the default from nvirt = 52 up
    // (below that the extra launches per slab cost more than the flops they save: measured crossover with
    // PPL_SYM_PAIR_SA at nocc = 5..8, nchol = 4 nvirt: 0.157 vs 0.186 ms at nvirt = 48, 0.283 vs 0.274 ms at 53,
    // 0.365 vs 0.328 ms at 64, 1.71 vs 0.97 ms at 96)
    full_plan(p, cap > p->ws_bytes ? cap - p->ws_bytes : 0);
    full_allocate(p);
    if (p->full_ok && nvirt >= full_min_v(p)) p->sym = PPL_SYM_FULL;
    return p;
}

int ppl_apply(ppl_plan_t *p, const double *L, const double *t2, double *R, void *stream) {
    return ppl_apply_ex(p, L, t2, R, nullptr, stream);
}

namespace {

// Launch-bound shapes: the whole ladder in one launch (ppl_kernels_small.cuh).  prof: an event pair around it.
int run_apply_small(ppl_plan_s *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts_in, cudaStream_t stream,
                    Prof *prof, bool fused_check = false) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, t2, R, &vec16);
    ppl_opts_t opts;
    if (rc == PPL_OK) rc = check_opts(opts_in, &opts);
    if (rc != PPL_OK) return fail(rc);
    static_assert(SMALL_SW_HOST == ppl::SMALL_SW, "planner and kernel disagree on the work item");
    if (prof && prof->mark(-1, 0, stream) != PPL_OK) return fail(PPL_ERR_CUDA);
    // bulk copies want 16-byte aligned rows of even length: otherwise (odd nvirt, t2 stored 'iajb', misaligned buffers) the
    // operands are first copied into the plan's padded buffers
    const int vp = p->vp, nb8 = (p->v + 7) / 8, ldt_pack = 8 * nb8 + ((nb8 & 1) ? 0 : 8);  // = ppl::SmallCfg<NB>::LDT
    const bool pack_L = (p->v & 1) || ((uintptr_t)L & 15), pack_t = (p->v & 1) || opts.t2_layout != PPL_LAYOUT_IJAB || ((uintptr_t)t2 & 15);
    if (pack_L || pack_t) {
        if (pack_L && !p->small_Lp && cudaMalloc(&p->small_Lp, (size_t)p->x * p->v * vp * 8) != cudaSuccess) {
            (void)cudaGetLastError();
            p->small_Lp = nullptr;
            return fail(PPL_ERR_ALLOC);
        }
        if (pack_t && !p->small_tp && cudaMalloc(&p->small_tp, (size_t)p->o * p->o * p->v * ldt_pack * 8) != cudaSuccess) {
            (void)cudaGetLastError();
            p->small_tp = nullptr;
            return fail(PPL_ERR_ALLOC);
        }
        const int64_t n = (pack_L ? (int64_t)p->x * p->v * vp : 0) + (pack_t ? (int64_t)p->o * p->o * p->v * ldt_pack : 0);
        const int g = (int)std::min<int64_t>((n + 255) / 256, (int64_t)p->num_sms * 8);
        ppl::k_small_prepack<<<g, 256, 0, stream>>>(pack_L ? L : nullptr, pack_t ? t2 : nullptr, p->small_Lp, p->small_tp, p->o, p->v, p->x,
                                                  vp, ldt_pack, r_strides(p->o, p->v, opts.t2_layout));
        PPL_CUDA(cudaGetLastError());
    }
    ppl::SmallArgs a;
    a.L = pack_L ? p->small_Lp : L;
    a.ldl = pack_L ? vp : p->v;
    a.t2 = pack_t ? p->small_tp : t2;
    a.ldt = pack_t ? ldt_pack : p->v;
    a.R = R;
    a.o = p->o;
    a.v = p->v;
    a.x = p->x;
    a.pair = p->sym != PPL_SYM_NONE ? 1 : 0;
    a.nitems = p->small_items[a.pair];
    a.alpha = opts.alpha;
    a.beta = opts.beta;
    a.rs = r_strides(p->o, p->v, opts.r_layout);
    a.chk.L = a.chk.t2 = nullptr;
    a.chk.flags = nullptr;
    a.ncheck = 0;
    a.seq = 0;
    a.done = p->vdone_dev;
    if (fused_check) {  // PPL_OPT_VERIFY_INPUTS = 1: the caller's t2, scanned by the first CTAs of the same launch.  Not L: this
                        // path never uses L[P,a,c] = L[P,c,a] (its result is right for any L), and scanning L -- 92 % of the
                        // check's bytes at `small` -- kept the check CTAs busy for the whole length of the kernel (ncu)
        a.chk.L = nullptr;
        a.chk.t2 = t2;
        a.chk.o = p->o;
        a.chk.v = p->v;
        a.chk.x = p->x;
        const ppl::RStrides ts = r_strides(p->o, p->v, opts.t2_layout);
        a.chk.s_i = ts.i;
        a.chk.s_j = ts.j;
        a.chk.s_c = ts.a;
        a.seq = ++p->vseq;
        const int slot = a.seq & 1;  // free: the caller has harvested everything but the newest outstanding check
        int *dflags = nullptr;
        PPL_CUDA(cudaHostGetDevicePointer(&dflags, p->vflags_host, 0));
        a.chk.flags = dflags + 8 + 8 * slot;
        a.done = p->vdone_dev + slot;
        p->vflags_host[8 + 8 * slot] = p->vflags_host[8 + 8 * slot + 1] = 0;
        const int nb = (p->v + 31) / 32;
        const int64_t items = (a.chk.L ? (int64_t)p->x * nb * (nb + 1) / 2 : 0) + (int64_t)p->o * (p->o + 1) / 2 * nb * nb;
        a.ncheck = (int)std::max<int64_t>(1, std::min<int64_t>(32, items / 4));
    }
    // every CTA of the grid is resident from the start (two per SM): a work-item CTA that had to wait for a check CTA's slot
    // would start its items late and end the kernel late (ncu: a check CTA scans its share of L for ~100 us at `small`)
    const int grid = std::min(a.nitems, 2 * p->num_sms - a.ncheck) + a.ncheck;
    // all of t2 staged once per CTA when every CTA has one work item and the region fits beside the ring (tiny: 80 KB)
    const size_t t2_region = ((size_t)p->o * p->o * p->v * a.ldt + (size_t)8 * nb8 * a.ldt + 8 * nb8) * 8;
    size_t smem_extra = 0;
    a.t2_resident = 0;
    a.nstages = ppl::SMALL_STAGES;
    const bool one_item = a.nitems + a.ncheck <= p->num_sms;  // one CTA per SM is enough: shared memory to spare
    if (one_item && t2_region <= (size_t)96 * 1024 && t2_region < ((size_t)1 << 20)) {
        a.t2_resident = 1;
        smem_extra = t2_region;
    }
    if (one_item) a.nstages = std::max(ppl::SMALL_STAGES, std::min(ppl::SMALL_MAX_STAGES, (p->x + ppl::BK - 1) / ppl::BK + 1));
    switch ((p->v + 7) / 8) {
#define PPL_LAUNCH_SMALL(NB)                                                                                    \
    case NB:                                                                                                    \
        while (a.nstages > ppl::SMALL_STAGES && ppl::SmallCfg<NB>::smem(a.nstages) + smem_extra > (size_t)200 * 1024) --a.nstages; \
        ppl::k_small_fused<NB><<<grid, ppl::SMALL_THREADS, ppl::SmallCfg<NB>::smem(a.nstages) + smem_extra, stream>>>(a); \
        break;
        PPL_LAUNCH_SMALL(1) PPL_LAUNCH_SMALL(2) PPL_LAUNCH_SMALL(3) PPL_LAUNCH_SMALL(4) PPL_LAUNCH_SMALL(5) PPL_LAUNCH_SMALL(6)
            PPL_LAUNCH_SMALL(7)
#undef PPL_LAUNCH_SMALL
        default: return fail(PPL_ERR_INVALID_ARG);
    }
    PPL_CUDA(cudaGetLastError());
    if (fused_check) {
        if (p->vq_n < 2) p->vq_seq[p->vq_n++] = a.seq;
        PPL_CUDA(cudaEventRecord(p->ev_vq[a.seq & 1], stream));
    }
    if (prof && prof->mark(K_STEP0, 1 + ((pack_L || pack_t) ? 1 : 0), stream) != PPL_OK) return fail(PPL_ERR_CUDA);
    return PPL_OK;
}

int apply_direct(ppl_plan_s *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts, cudaStream_t stream) {
    if (p && p->small_ok) return run_apply_small(p, L, t2, R, opts, stream, nullptr);
    if (p && p->sym == PPL_SYM_FULL) return run_apply_full(p, L, t2, R, opts, stream, nullptr);
    return run_apply(p, L, t2, R, opts, stream, nullptr);
}

// Launch-bound shapes (tiny: 6 launches of a few microseconds; small: 33 launches, 4 side streams and
// ~60 event operations for 46 us of DMMA work): the whole apply -- forks and joins of the side streams
// included -- is captured once into a CUDA graph, keyed on the three pointers, the options and the
// symmetry mode, and replayed with one cudaGraphLaunch while the key stays the same (a CCSD iteration
// calls the ladder on the same buffers).  A new key re-captures (the TMA descriptors of L and t2 are
// kernel parameters, so the nodes cannot simply be re-pointed).
int apply_graph(ppl_plan_s *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts_in, cudaStream_t stream) {
    ppl_opts_t opts;
    bool vec16;
    int rc = check_ptrs(p, L, t2, R, &vec16);
    if (rc == PPL_OK) rc = check_opts(opts_in, &opts);
    if (rc != PPL_OK) return fail(rc);
    const ppl_plan_s::GraphKey &k = p->gkey;
    const bool hit = p->gexec && k.L == L && k.t2 == t2 && k.R == R && k.sym == p->sym && k.opts.t2_layout == opts.t2_layout &&
                     k.opts.r_layout == opts.r_layout && k.opts.alpha == opts.alpha && k.opts.beta == opts.beta;
    if (!hit) {
        if (p->gexec) {
            cudaGraphExecDestroy(p->gexec);
            p->gexec = nullptr;
        }
        if (!p->gcap) PPL_CUDA(cudaStreamCreateWithFlags(&p->gcap, cudaStreamNonBlocking));
        PPL_CUDA(cudaStreamBeginCapture(p->gcap, cudaStreamCaptureModeRelaxed));
        rc = apply_direct(p, L, t2, R, &opts, p->gcap);
        cudaGraph_t g = nullptr;
        const cudaError_t e = cudaStreamEndCapture(p->gcap, &g);  // also ends a capture that failed half way
        if (rc != PPL_OK || e != cudaSuccess || !g) {
            if (g) cudaGraphDestroy(g);
            (void)cudaGetLastError();
            return rc != PPL_OK ? rc : fail(PPL_ERR_CUDA);
        }
        const cudaError_t ei = cudaGraphInstantiate(&p->gexec, g, 0);
        cudaGraphDestroy(g);
        if (ei != cudaSuccess) {
            (void)cudaGetLastError();
            p->gexec = nullptr;
            return fail(PPL_ERR_CUDA);
        }
        p->gkey.L = L;
        p->gkey.t2 = t2;
        p->gkey.R = R;
        p->gkey.opts = opts;
        p->gkey.sym = p->sym;
    }
    PPL_CUDA(cudaGraphLaunch(p->gexec, stream));
    return PPL_OK;
}

}  // namespace

int ppl_apply_ex(ppl_plan_t *p, const double *L, const double *t2, double *R, const ppl_opts_t *opts, void *stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (!p || !L || !t2 || !R || !device_ok(p)) return fail(PPL_ERR_INVALID_ARG);
    // a caller who is capturing `stream` gets the plain launches recorded into their own graph (and no input check:
    // its result could not be read back during the capture)
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &st) != cudaSuccess) {
        (void)cudaGetLastError();
        st = cudaStreamCaptureStatusActive;
    }
    if (st == cudaStreamCaptureStatusNone) {
        int rc = verify_harvest(p, nullptr, false);  // what the previous apply's check found
        if (rc != PPL_OK) return rc;
        if (p->verify && p->sym != PPL_SYM_NONE) {
            // launch-bound shapes: the check rides in the apply's one launch (its first CTAs) instead of a launch of its own
            if (p->verify == 1 && p->small_ok) return run_apply_small(p, L, t2, R, opts, stream, nullptr, true);
            ppl_opts_t o;
            if (check_opts(opts, &o) != PPL_OK) return fail(PPL_ERR_INVALID_ARG);
            // PPL_SYM_FULL, mode 1: the check (HBM-bound: it reads L and t2 once) runs on the plan's producer stream, which that
            // mode leaves idle, beside the first slab's step 0 instead of in front of it; `stream` joins it at the end of the
            // apply, so that nothing queued later can change the inputs under it
            const bool aside = p->sym == PPL_SYM_FULL && p->verify == 1 && p->gen != nullptr;
            if (aside) {
                PPL_CUDA(cudaEventRecord(p->ev_in, stream));
                PPL_CUDA(cudaStreamWaitEvent(p->gen, p->ev_in, 0));
            }
            rc = verify_begin(p, p->sym == PPL_SYM_FULL ? L : nullptr, t2, o.t2_layout, aside ? p->gen : stream);
            if (rc != PPL_OK) return rc;
            if (aside) {
                rc = graph_wanted(p) ? apply_graph(p, L, t2, R, opts, stream) : apply_direct(p, L, t2, R, opts, stream);
                PPL_CUDA(cudaStreamWaitEvent(stream, p->ev_verify, 0));
                return rc;
            }
        }
        if (graph_wanted(p)) return apply_graph(p, L, t2, R, opts, stream);
    }
    return apply_direct(p, L, t2, R, opts, stream);
}

int ppl_apply_profiled(ppl_plan_t *p, const double *L, const double *t2, double *R, void *stream_, ppl_times_t *times) {
    if (!times) return fail(PPL_ERR_INVALID_ARG);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    memset(times, 0, sizeof(*times));
    Prof prof;
    int rc = (p && p->small_ok) ? run_apply_small(p, L, t2, R, nullptr, stream, &prof)
             : (p && p->sym == PPL_SYM_FULL) ? run_apply_full(p, L, t2, R, nullptr, stream, &prof)
                                             : run_apply(p, L, t2, R, nullptr, stream, &prof);
    const cudaError_t e = cudaStreamSynchronize(stream);
    if (rc == PPL_OK && e == cudaSuccess && prof.ev.size() >= 2) {
        float acc[K_KINDS] = {0, 0, 0, 0, 0};
        for (size_t k = 1; k < prof.ev.size(); ++k) {
            float ms = 0;
            cudaEventElapsedTime(&ms, prof.ev[k - 1], prof.ev[k]);
            if (prof.kind[k] >= 0) acc[prof.kind[k]] += ms;
        }
        cudaEventElapsedTime(&times->total_ms, prof.ev.front(), prof.ev.back());
        times->pack_ms = acc[K_PACK];
        times->step0_ms = acc[K_STEP0];
        times->fold_ms = acc[K_FOLD];
        times->step1_ms = acc[K_STEP1];
        times->reduce_ms = acc[K_REDUCE];
        times->n_pack = prof.launches[K_PACK];
        times->n_step0 = prof.launches[K_STEP0];
        times->n_fold = prof.launches[K_FOLD];
        times->n_step1 = prof.launches[K_STEP1];
        times->n_reduce = prof.launches[K_REDUCE];
    }
    for (auto &x : prof.ev) cudaEventDestroy(x);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(PPL_ERR_CUDA);
    }
    return rc;
}

int ppl_apply_dense(ppl_plan_t *p, const double *eri, int a0, int na, const double *t2, double *R, const ppl_opts_t *opts_in,
                    void *stream_) {
    bool vec16 = false;
    int rc = check_ptrs(p, eri, t2, R, &vec16);
    ppl_opts_t opts;
    if (rc == PPL_OK) rc = check_opts(opts_in, &opts);
    if (rc == PPL_OK && (a0 < 0 || na < 1 || a0 + na > p->v)) rc = PPL_ERR_INVALID_ARG;
    if (rc != PPL_OK) return fail(rc);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    const double *t2m = t2;
    if ((rc = t2_matrix(p, t2, opts.t2_layout, stream, &t2m)) != PPL_OK) return rc;
    const bool tma = p->use_tma && vec16;
    const int M = p->o * p->o;
    const int64_t rows = (int64_t)na * p->v;
    CUtensorMap mapT, mapE;
    if (tma && (make_map_2d(&mapT, t2m, (uint64_t)p->vv, (uint64_t)M, (uint64_t)p->vv * 8, ppl::BK, (uint32_t)p->bm_full) != PPL_OK ||
                make_map_2d(&mapE, eri, (uint64_t)p->vv, (uint64_t)rows, (uint64_t)p->vv * 8, ppl::BK, ppl::BN) != PPL_OK))
        return fail(PPL_ERR_CUDA);
    // rows of the slab matrix [(a,b)][(c,d)] in chunks the partials buffer can hold
    // (the buffer was sized for N <= T*T rows at the planner's split: with split-K 1 it holds part_bytes / (8 M) rows)
    int64_t chunk = std::min<int64_t>(rows, (int64_t)(p->part_bytes / ((size_t)8 * M)));
    if (chunk >= ppl::BN) chunk = chunk / ppl::BN * ppl::BN;
    if (chunk < 1) return fail(PPL_ERR_WORKSPACE_TOO_SMALL);
    Tile t;
    t.a0 = a0;
    t.b0 = 0;
    t.ta = na;
    t.tb = p->v;
    t.mirror = 0;
    for (int64_t n0 = 0; n0 < rows; n0 += chunk) {
        const int N = (int)std::min<int64_t>(chunk, rows - n0);
        SplitChoice sc = choose_split(M, N, p->vv, p->num_sms, p->mg_full, p->part_bytes);
        if ((size_t)sc.splitk * M * N * 8 > p->part_bytes) return fail(PPL_ERR_WORKSPACE_TOO_SMALL);
        const double *B = eri + n0 * p->vv;
        CUtensorMap mapB;  // the chunk's rows as their own tensor so that tile-edge rows beyond it read as zero
        if (tma && make_map_2d(&mapB, B, (uint64_t)p->vv, (uint64_t)N, (uint64_t)p->vv * 8, ppl::BK, ppl::BN) != PPL_OK)
            return fail(PPL_ERR_CUDA);
        rc = launch_step1(p, tma ? &mapT : nullptr, tma ? &mapB : nullptr, p->mg_full, t2m, p->vv, B, p->vv, M, N, p->vv, sc,
                          p->part, vec16, stream);
        if (rc == PPL_OK) rc = launch_reduce(p, t, sc.splitk, N, (int)n0, p->v, R, opts, stream);
        if (rc != PPL_OK) return rc;
    }
    (void)mapE;
    return PPL_OK;
}

// Step 0 alone: the dense slab eri[a - a0][b][c][d] = <ab|cd> = sum_P L[P,a,c] L[P,b,d] for a0 <= a < a0 + na, all b, c, d.
// One W tile (A-block = the slab, B-block = all b) written straight into the caller's buffer: its [(a,b)][(c,d)] row
// order IS the paper's 'abcd'.  Slabs are cut into pieces of at most 64 a's so that a piece is one grouped raster.
int ppl_generate_eri(ppl_plan_t *p, const double *L, int a0, int na, double *eri, void *stream_) {
    bool vec16 = false;
    int rc = check_ptrs(p, L, L, eri, &vec16);
    if (rc == PPL_OK && (a0 < 0 || na < 1 || a0 + na > p->v)) rc = PPL_ERR_INVALID_ARG;
    if (rc != PPL_OK) return fail(rc);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    const bool tma = p->use_tma && vec16;
    CUtensorMap mapL;
    if (tma && make_map_2d(&mapL, L, (uint64_t)p->vv, (uint64_t)p->x, (uint64_t)p->vv * 8, 16, ppl::BK) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    for (int a = a0; a < a0 + na; a += 64) {
        Tile t;
        t.a0 = a;
        t.ta = std::min(64, a0 + na - a);
        t.b0 = 0;
        t.tb = p->v;
        t.mirror = 0;
        double *W = eri + (int64_t)(a - a0) * p->v * p->vv;
        if ((rc = launch_step0(p, t, L, tma ? &mapL : nullptr, W, vec16, stream)) != PPL_OK) return rc;
    }
    return PPL_OK;
}

}  // extern "C"

namespace {

// hflags: two words of the plan's mapped pinned host buffer; cleared here by the host, written by the kernel (no memset, no
// device-to-host copy: at launch-bound shapes those two operations cost more than the check itself)
int launch_check(const ppl_plan_s *p, const double *L, const double *t2, int t2_layout, int *hflags, cudaStream_t stream) {
    ppl::CheckArgs a;
    a.L = L;
    a.t2 = t2;
    a.o = p->o;
    a.v = p->v;
    a.x = p->x;
    const ppl::RStrides ts = r_strides(p->o, p->v, t2_layout);
    a.s_i = ts.i;
    a.s_j = ts.j;
    a.s_c = ts.a;
    int *dflags = nullptr;
    PPL_CUDA(cudaHostGetDevicePointer(&dflags, hflags, 0));
    a.flags = dflags;
    hflags[0] = hflags[1] = 0;
    const int nb = (p->v + 31) / 32;
    const int64_t items = (L ? (int64_t)p->x * nb * (nb + 1) / 2 : 0) + (t2 ? (int64_t)p->o * (p->o + 1) / 2 * nb * nb : 0);
    ppl::k_check_inputs<<<(int)std::max<int64_t>(1, std::min<int64_t>(items, (int64_t)p->num_sms * 8)), 256, 0, stream>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// Result of the outstanding per-apply verifications.  A k_check_inputs launch (the tiled paths): waits for that head-of-apply
// kernel only.  The check CTAs of k_small_fused (launch-bound shapes): the last of them stores the apply's sequence number into
// mapped host memory; wait_all = false (the head of the next apply) does not wait for the NEWEST of them -- that apply may
// still be running, and waiting would serialise the host with the device (tiny: 25 instead of 18 us per back-to-back apply)
// -- but reads it if it is there, and waits for an older one; so a violation is reported by the next call or the one after.
// Should a launch have died its number never arrives: every so often ask the event recorded behind that launch (on whichever
// stream the caller gave for it), and stop once it has completed.
int verify_harvest(ppl_plan_s *p, int *flags_out, bool wait_all) {
    if (flags_out) *flags_out = 0;
    int h = 0;
    bool any = false;
    if (p->verify_pending) {
        p->verify_pending = 0;
        if (cudaEventSynchronize(p->ev_verify) != cudaSuccess) {
            (void)cudaGetLastError();
            return fail(PPL_ERR_CUDA);
        }
        h |= (p->vflags_host[0] ? 1 : 0) | (p->vflags_host[1] ? 2 : 0);
        any = true;
    }
    while (p->vq_n > 0) {
        const int seq = p->vq_seq[0], slot = seq & 1;
        volatile int *w = p->vflags_host + 8 + 8 * slot;
        const bool must = wait_all || p->vq_n > 1;
        if (!must && w[4] != seq) break;
        for (unsigned spin = 1; w[4] != seq; ++spin) {
            if ((spin & 0x3ff) == 0) {
                const cudaError_t e = cudaEventQuery(p->ev_vq[slot]);  // complete <=> the launch of this check has left the GPU
                if (e == cudaErrorNotReady) continue;
                if (e != cudaSuccess || w[4] != seq) {
                    (void)cudaGetLastError();
                    p->vq_n = 0;
                    return fail(PPL_ERR_CUDA);
                }
            }
        }
        h |= (w[0] ? 1 : 0) | (w[1] ? 2 : 0);
        any = true;
        p->vq_seq[0] = p->vq_seq[1];
        --p->vq_n;
    }
    if (!any) return PPL_OK;
    if (flags_out) *flags_out = h;
    if ((h & 2) && p->sym != PPL_SYM_NONE) return fail(PPL_ERR_PRECONDITION);
    if ((h & 1) && p->sym == PPL_SYM_FULL) return fail(PPL_ERR_PRECONDITION);
    return PPL_OK;
}

// queue the check of this apply's inputs on `stream` (L == nullptr / t2 == nullptr: not checked)
int verify_begin(ppl_plan_s *p, const double *L, const double *t2, int t2_layout, cudaStream_t stream) {
    int rc = launch_check(p, L, t2, t2_layout, p->vflags_host, stream);
    if (rc != PPL_OK) return rc;
    PPL_CUDA(cudaEventRecord(p->ev_verify, stream));
    p->verify_pending = 1;
    if (p->verify == 2) return verify_harvest(p, nullptr);
    return PPL_OK;
}

}  // namespace

extern "C" {

int ppl_check_inputs(ppl_plan_t *p, const double *L, const double *t2, void *stream_, int *flags) {
    if (!p || !L || !t2 || !device_ok(p)) return fail(PPL_ERR_INVALID_ARG);
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    const int rc = launch_check(p, L, t2, PPL_LAYOUT_IJAB, p->vflags_host + 2, stream);
    if (rc != PPL_OK) return rc;
    PPL_CUDA(cudaStreamSynchronize(stream));
    const int h = (p->vflags_host[2] ? 1 : 0) | (p->vflags_host[3] ? 2 : 0);
    if (flags) *flags = h;
    if ((h & 2) && p->sym != PPL_SYM_NONE) return fail(PPL_ERR_PRECONDITION);
    if ((h & 1) && p->sym == PPL_SYM_FULL) return fail(PPL_ERR_PRECONDITION);
    return PPL_OK;
}

int ppl_plan_verify_status(ppl_plan_t *p, int *flags) {
    if (!p) return fail(PPL_ERR_INVALID_ARG);
    return verify_harvest(p, flags);
}

}  // extern "C"

// ---- what ppl_host.cu calls (ppl_launch.h) ----
namespace pplapi {

int map_2d(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t row_bytes, uint32_t box_inner,
           uint32_t box_outer) {
    return make_map_2d(map, base, inner, outer, row_bytes, box_inner, box_outer);
}

int step0_tile(const ppl_plan_s *p, const Tile &t, const CUtensorMap *mapA, int a0v, const CUtensorMap *mapB, int b0v, double *W,
               cudaStream_t s) {
    ppl::Step0TmaArgs a;
    a.a0v = a0v;
    a.b0v = b0v;
    a.M = t.ta * p->v;
    a.N = t.tb * p->v;
    a.K = p->x;
    a.v = p->v;
    a.tb = t.tb;
    a.W = W;
    a.ldw = p->vv;
    const int items = ((a.M + ppl::BM - 1) / ppl::BM) * ((a.N + ppl::BN - 1) / ppl::BN);
    ppl::k_step0_tma<<<std::min(items, p->num_sms), ppl::TMA_THREADS, ppl::SMEM_TMA, s>>>(*mapA, *mapB, a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

uint32_t step1_box_rows(const ppl_plan_s *p) { return (uint32_t)p->bm_full; }

int step1_tile(const ppl_plan_s *p, const CUtensorMap *mapT, const double *t2, int slot, const Tile &t, cudaStream_t s) {
    return launch_step1(p, mapT, &p->mapW[slot], p->mg_full, t2, p->vv, p->slot[slot], p->vv, p->o * p->o, t.ta * t.tb, p->vv, t.full,
                        p->part, true, s);
}

int reduce_tile(const ppl_plan_s *p, const Tile &t, double *R, int64_t si, int64_t sj, int64_t sa, int64_t sb, double alpha,
                double beta, cudaStream_t s, int64_t r_bias) {
    ppl::ReduceArgs a;
    a.part = p->part;
    a.splitk = t.full.splitk;
    a.M = p->o * p->o;
    a.N = t.ta * t.tb;
    a.o = p->o;
    a.v = p->v;
    a.tb = t.tb;
    a.a0 = t.a0;
    a.b0 = t.b0;
    a.n_off = 0;
    a.mirror = t.mirror;
    a.alpha = alpha;
    a.beta = beta;
    a.rs.i = si;
    a.rs.j = sj;
    a.rs.a = sa;
    a.rs.b = sb;
    a.R = R;
    a.r_bias = r_bias;
    const int64_t MN = (int64_t)a.M * a.N;
    const int grid = (int)std::min<int64_t>((MN + 255) / 256, (int64_t)p->num_sms * 8);
    ppl::k_reduce<<<grid, 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int pack_rows(const ppl_plan_s *p, const double *chunk, double diag, cudaStream_t s, int row0, int row1) {
    return launch_pack(p, chunk, PPL_LAYOUT_IJAB, diag, s, row0, row1, (int64_t)row0 * p->vv);
}

// rows [row0, row1) of t2 (the staged chunk, row row0 first) against the tau+- rows their mirror images wrote:
// sets bit 1 of the per-apply verification flags (the words verify_begin cleared), see k_check_t2_rows
int check_rows(const ppl_plan_s *p, const double *chunk, double diag, cudaStream_t s, int row0, int row1) {
    ppl::CheckRowsArgs a;
    a.t2 = chunk;
    a.taup = p->taup;
    a.taum = p->taum;
    a.ldp = p->ldp;
    a.ldm = p->ldm;
    a.row0 = row0;
    a.row1 = row1;
    a.o = p->o;
    a.v = p->v;
    a.vp = p->vp;
    a.scale = 0.5;
    a.diag = diag;
    int *dflags = nullptr;
    PPL_CUDA(cudaHostGetDevicePointer(&dflags, p->vflags_host, 0));
    a.flags = dflags;
    const int nb = (p->v + 31) / 32;
    const int64_t items = (int64_t)(row1 - row0) * nb * (nb + 1) / 2;
    ppl::k_check_t2_rows<<<(int)std::max<int64_t>(1, std::min<int64_t>(items, (int64_t)p->num_sms * 8)), 256, 0, s>>>(a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

int unpack_range(const ppl_plan_s *p, double *R, int64_t idx0, int64_t idx1, cudaStream_t s) {
    ppl_opts_t opts;
    check_opts(nullptr, &opts);
    return launch_unpack_full(p, opts, R, idx0, idx1, s);
}

int full_compute(ppl_plan_s *p, const double *L, cudaStream_t s, cudaEvent_t tau_ready, const SlabHook *hook) {
    return run_apply_full(p, L, nullptr, nullptr, nullptr, s, nullptr, FULL_COMPUTE, tau_ready, hook);
}

int unpack_slab(const ppl_plan_s *p, double *slab, int a0, int na, cudaStream_t s) {
    ppl_opts_t opts;
    check_opts(nullptr, &opts);
    ppl::RStrides rs;  // the slab buffer holds R[i][j][a - a0][b], dense
    rs.i = (int64_t)p->o * na * p->v;
    rs.j = (int64_t)na * p->v;
    rs.a = p->v;
    rs.b = 1;
    return launch_unpack_full(p, opts, slab, 0, (int64_t)p->o * p->o * na * p->v, s, a0, na, &rs, (int64_t)a0 * rs.a);
}

int verify_begin(ppl_plan_s *p, const double *L, const double *t2, int t2_layout, cudaStream_t stream) {
    return ::verify_begin(p, L, t2, t2_layout, stream);
}
int verify_harvest(ppl_plan_s *p, int *flags_out) { return ::verify_harvest(p, flags_out, true); }

}  // namespace pplapi

// ---- plain GEMMs on the TMA kernels, for ppl_contract_pair's fast paths (ppl_internal.h) ----
// C[M][N] (dense) = beta C + alpha A^T B with A[K][M], B[K][N] dense row-major ("k-outer": 'k..m..,k..n..->m..n..'): k_step0_tma
int ppl_gemm_kouter_tma(const double *A, const double *B, int M, int N, int K, double *C, double alpha, double beta, int sms,
                        cudaStream_t s) {
    if (set_kernel_attrs() != PPL_OK) return fail(PPL_ERR_CUDA);
    CUtensorMap mapA, mapB;
    if (make_map_2d(&mapA, A, (uint64_t)M, (uint64_t)K, (uint64_t)M * 8, 16, ppl::BK) != PPL_OK ||
        make_map_2d(&mapB, B, (uint64_t)N, (uint64_t)K, (uint64_t)N * 8, 16, ppl::BK) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    ppl::Step0TmaArgs a;
    a.a0v = a.b0v = 0;
    a.M = M;
    a.N = N;
    a.K = K;
    a.v = N;  // with tb = 1 and ldw = N^2 the kernel's store address is m N + n (ppl_kernels_tma.cuh)
    a.tb = 1;
    a.W = C;
    a.ldw = (int64_t)N * N;
    a.alpha = alpha;
    a.beta = beta;
    const int64_t items = (int64_t)((M + ppl::BM - 1) / ppl::BM) * ((N + ppl::BN - 1) / ppl::BN);
    ppl::k_step0_tma<<<(int)std::min<int64_t>(items, sms), ppl::TMA_THREADS, ppl::SMEM_TMA, s>>>(mapA, mapB, a);
    PPL_CUDA(cudaGetLastError());
    return PPL_OK;
}

// part[z][M][N] = sum_{k in split z} A[m][k] B[n][k] with A[M][K], B[N][K] dense row-major ("k-inner"): k_step1_tma.
// part_bytes: room for the partials; *splitk_out: the split taken (>= 1).  PPL_ERR_WORKSPACE_TOO_SMALL if M N doubles do not fit.
int ppl_gemm_kinner_tma(const double *A, const double *B, int M, int N, int K, double *part, size_t part_bytes, int *splitk_out,
                        int sms, cudaStream_t s) {
    if (set_kernel_attrs() != PPL_OK) return fail(PPL_ERR_CUDA);
    if ((size_t)M * N * 8 > part_bytes) return fail(PPL_ERR_WORKSPACE_TOO_SMALL);
    const MGeom mg = m_geom_tma(M, 10);
    const SplitChoice sc = choose_split(M, N, K, sms, mg, part_bytes);
    CUtensorMap mapA, mapB;
    if (make_map_2d(&mapA, A, (uint64_t)K, (uint64_t)M, (uint64_t)K * 8, ppl::BK, (uint32_t)(16 * mg.ni)) != PPL_OK ||
        make_map_2d(&mapB, B, (uint64_t)K, (uint64_t)N, (uint64_t)K * 8, ppl::BK, ppl::BN) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    ppl_plan_s tmp;  // launch_step1 reads the SM count only
    tmp.num_sms = sms;
    const int rc = launch_step1(&tmp, &mapA, &mapB, mg, A, K, B, K, M, N, K, sc, part, true, s);
    if (splitk_out) *splitk_out = sc.splitk;
    return rc;
}

extern "C" {

int ppl_destroy(ppl_plan_t *p) {
    if (!p) return PPL_OK;
    const int rc = p->dry ? PPL_OK : verify_harvest(p, nullptr);  // a violation found by the last apply's check is not lost
    free_plan(p);
    return rc;
}

int ppl_probe_fp64_pipe(int kind, double *tflops, int reps, double ms_target) {
    if (!tflops || reps < 1 || kind < PPL_PROBE_DMMA8 || kind > PPL_PROBE_MIX8) return fail(PPL_ERR_INVALID_ARG);
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
    const int sms = prop.multiProcessorCount, threads = 512, warps = threads / 32;
    // flops per loop iteration of one warp: a DMMA m8n8k4 is 8*8*4*2 = 512, a DFMA 2 per lane
    double per_warp = 0;
    switch (kind) {
        case PPL_PROBE_DMMA8: per_warp = 8 * 512.0; break;
        case PPL_PROBE_DMMA16: per_warp = 16 * 512.0; break;
        case PPL_PROBE_DFMA16: per_warp = 16 * 64.0; break;
        case PPL_PROBE_MIX8: per_warp = 8 * (512.0 + 64.0); break;
    }
    const double flop_per_iter = per_warp * warps * sms;
    const int iters = (int)std::max(1024.0, ms_target * 1e-3 * PEAK_FLOPS / flop_per_iter);
    double best = 0;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0, 0);
        switch (kind) {
            case PPL_PROBE_DMMA8: ppl::k_probe_dmma<<<sms, threads>>>(out, iters, 1.0000001, 1e-9); break;
            case PPL_PROBE_DMMA16: ppl::k_probe_dmma_n<16><<<sms, threads>>>(out, iters, 1.0000001, 1e-9); break;
            case PPL_PROBE_DFMA16: ppl::k_probe_dfma<16><<<sms, threads>>>(out, iters, 1.0000001, 1e-9); break;
            case PPL_PROBE_MIX8: ppl::k_probe_mix<8><<<sms, threads>>>(out, iters, 1.0000001, 1e-9); break;
        }
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

int ppl_probe_fp64_peak(double *tflops, int reps, double ms_target) {
    return ppl_probe_fp64_pipe(PPL_PROBE_DMMA8, tflops, reps, ms_target);
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
