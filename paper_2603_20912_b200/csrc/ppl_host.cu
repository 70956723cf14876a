// ppl_host.cu -- ppl_apply_host: the ladder on HOST-resident operands (the paper's own setting: operands in host memory,
// PAPER.md:85, 146-181).  Copies and their overlap with the kernels live here; every launch goes
// through ppl_api.cu (ppl_launch.h), where the kernels are instantiated.
//   PPL_SYM_FULL            apply_host_full:   t2 and R streamed in (i,j) chunks through two staging buffers, L whole
//   PPL_SYM_NONE / PAIR     apply_host_tiles:  t2 resident, L whole or as row panels, R as slabs (NONE) or resident (PAIR)
//   otherwise               everything copied whole around ppl_apply
#include "../../include/ppl.h"
#include "ppl_launch.h"

#include <algorithm>
#include <cstdint>
#include <initializer_list>

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

bool dev_alloc(double **ptr, size_t bytes) {
    if (*ptr) return true;
    if (cudaMalloc(ptr, bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        *ptr = nullptr;
        return false;
    }
    return true;
}
void dev_free(double **ptr) {
    if (*ptr) cudaFree(*ptr);
    *ptr = nullptr;
}
}  // namespace

static int host_events(ppl_plan_s *p);

// PPL_SYM_FULL on host operands: the device never holds t2 or R.  t2 is streamed through two staging buffers and
// packed chunk by chunk into tau+- (rows (i,j) of a chunk are contiguous in the [i][j][c][d] order), the slabs run on
// the packed operands, and R leaves slab by slab WHILE they run: the rows a of R[i,j,a,b] that belong to a slab of the loop
// are final as soon as that slab's reductions are (k_unpack_full on the a-range: slab R[:, :, A, :] in by a 2-D copy,
// R += term, slab out), so that at the end only the last, smallest slab is still to travel.
// Device residency: L + tau+- + R+-acc + the PPL_SYM_FULL workspace -- about half of L + t2 + R + workspace, which
// is what lets the paper's Table 3 shapes (t2 and R of 39 GB each at N = 800) run on one 180 GB GPU.
struct FullHostCtx {
    ppl_plan_s *p;
    double *Rh;
    cudaStream_t st[2];
    int k;
};
// called behind the launches of every slab (ppl_launch.h, SlabHook): the R+-acc columns of the a's [a0, a0 + ta) are final
// once the work queued so far on s_plus / s_minus has run
static int full_slab_hook(void *ctx_, int a0, int ta, cudaStream_t s_plus, cudaStream_t s_minus) {
    FullHostCtx &c = *static_cast<FullHostCtx *>(ctx_);
    ppl_plan_s *p = c.p;
    ppl_plan_s::HostStream &h = p->hsn;
    const int na = std::min(ta, p->v - a0);  // (odd nvirt: the pad index of the packed geometry is no row of R)
    if (na <= 0) return PPL_OK;
    const int slot = c.k & 1;
    cudaStream_t s = c.st[slot];
    ++c.k;
    const size_t w = (size_t)na * p->v * 8, pitch = (size_t)p->vv * 8, rows = (size_t)p->o * p->o;
    PPL_CUDA(cudaMemcpy2DAsync(h.rs[slot], w, c.Rh + (size_t)a0 * p->v, pitch, w, rows, cudaMemcpyHostToDevice, s));
    PPL_CUDA(cudaEventRecord(h.ev_rsdone[slot], s_plus));
    PPL_CUDA(cudaStreamWaitEvent(s, h.ev_rsdone[slot], 0));
    if (s_minus != s_plus) {
        PPL_CUDA(cudaEventRecord(h.ev_rsin[slot], s_minus));
        PPL_CUDA(cudaStreamWaitEvent(s, h.ev_rsin[slot], 0));
    }
    const int rc = pplapi::unpack_slab(p, h.rs[slot], a0, na, s);
    if (rc != PPL_OK) return rc;
    PPL_CUDA(cudaMemcpy2DAsync(c.Rh + (size_t)a0 * p->v, pitch, h.rs[slot], w, w, rows, cudaMemcpyDeviceToHost, s));
    return PPL_OK;
}

static int apply_host_full_queue(ppl_plan_s *p, const double *Lh, const double *t2h, double *Rh, uint64_t *h2d, uint64_t *d2h) {
    const size_t nL = (size_t)p->x * p->vv * 8;
    const int64_t rows = (int64_t)p->o * p->o;
    const size_t row_bytes = (size_t)p->vv * 8;
    if (!p->dL && cudaMalloc(&p->dL, nL) != cudaSuccess) {
        (void)cudaGetLastError();
        p->dL = nullptr;
        return fail(PPL_ERR_ALLOC);
    }
    if (!p->hstage[0]) {
        const size_t want = p->dbg.host_chunk_mb > 0 ? (size_t)p->dbg.host_chunk_mb << 20 : (size_t)1 << 30;  // debug override of the staging-buffer size
        p->hchunk_rows = (int)std::max<int64_t>(1, std::min<int64_t>(rows, (int64_t)(want / row_bytes)));
        for (int i = 0; i < 2; ++i)
            if (cudaMalloc(&p->hstage[i], (size_t)p->hchunk_rows * row_bytes) != cudaSuccess) {
                (void)cudaGetLastError();
                for (int k = 0; k < 2; ++k) {
                    if (p->hstage[k]) cudaFree(p->hstage[k]);
                    p->hstage[k] = nullptr;
                }
                return fail(PPL_ERR_ALLOC);
            }
    }
    if (!p->hs2) {
        bool ok = cudaStreamCreateWithFlags(&p->hs2, cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&p->ev_tau, cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) {
            (void)cudaGetLastError();
            return fail(PPL_ERR_CUDA);
        }
    }
    {
        int rce = host_events(p);
        if (rce != PPL_OK) return rce;
        ppl_plan_s::HostStream &h = p->hsn;
        const size_t slab = (size_t)rows * ppl::TA_FULL * p->v * 8;  // R[:, :, 16 a's, :]
        if (h.slab_bytes < slab) {
            for (int i = 0; i < 2; ++i) dev_free(&h.rs[i]);
            h.slab_bytes = slab;
        }
        if (!dev_alloc(&h.rs[0], h.slab_bytes) || !dev_alloc(&h.rs[1], h.slab_bytes)) {
            for (int i = 0; i < 2; ++i) dev_free(&h.rs[i]);
            h.slab_bytes = 0;
            return fail(PPL_ERR_ALLOC);
        }
    }
    cudaStream_t cs = p->host_stream;         // L in, all slabs
    cudaStream_t st[2] = {p->gen, p->hs2};    // chunk k of t2, then slab k of R, on stream k % 2; each stream owns one buffer of each kind
    const bool minus = p->Mm > 0 && p->Km > 0;
    // phase A: L in on the compute stream; t2 chunks in -> tau+- on the chunk streams, overlapping L and step 0 of slab 0
    PPL_CUDA(cudaMemcpyAsync(p->dL, Lh, nL, cudaMemcpyHostToDevice, cs));
    if (p->verify) {  // L here; t2 never sits on the device whole and is verified chunk by chunk below (same flag words)
        const int rcv = pplapi::verify_begin(p, p->dL, nullptr, PPL_LAYOUT_IJAB, cs);
        if (rcv != PPL_OK) return rcv;
    }
    PPL_CUDA(cudaMemsetAsync(p->raccp, 0, (size_t)p->Mp * p->ldp * 8, cs));
    if (minus) PPL_CUDA(cudaMemsetAsync(p->raccm, 0, (size_t)p->Mm * p->ldm * 8, cs));
    int k = 0;
    for (int64_t r0 = 0; r0 < rows; r0 += p->hchunk_rows, ++k) {
        const int64_t r1 = std::min<int64_t>(rows, r0 + p->hchunk_rows);
        cudaStream_t s = st[k & 1];
        double *buf = p->hstage[k & 1];
        PPL_CUDA(cudaMemcpyAsync(buf, t2h + r0 * p->vv, (size_t)(r1 - r0) * row_bytes, cudaMemcpyHostToDevice, s));
        int rc = pplapi::pack_rows(p, buf, 0.5, s, (int)r0, (int)r1);
        if (rc != PPL_OK) return rc;
        if (p->verify) {
            // pair symmetry of t2: the rows i >= j of the chunk against the tau+- rows their mirror images (j,i) <= (i,j)
            // wrote -- in this chunk, in chunk k - 2, k - 4, ... (this stream) or in chunk k - 1, k - 3, ... (the other one)
            PPL_CUDA(cudaEventRecord(p->hsn.ev_chunk[k & 1], s));
            if (k > 0) PPL_CUDA(cudaStreamWaitEvent(s, p->hsn.ev_chunk[(k - 1) & 1], 0));
            rc = pplapi::check_rows(p, buf, 0.5, s, (int)r0, (int)r1);
            if (rc != PPL_OK) return rc;
        }
    }
    PPL_CUDA(cudaEventRecord(p->ev_in, st[1]));
    PPL_CUDA(cudaStreamWaitEvent(st[0], p->ev_in, 0));
    PPL_CUDA(cudaEventRecord(p->ev_tau, st[0]));
    // phase B: all slabs on the packed operands; behind every slab its rows of R travel in, take the term and travel out
    // (slab k on chunk stream k & 1, which owns slab buffer k & 1: in order, so a buffer is refilled behind its D2H copy)
    FullHostCtx ctx{p, Rh, {st[0], st[1]}, 0};
    const pplapi::SlabHook hook{full_slab_hook, &ctx};
    int rc = pplapi::full_compute(p, p->dL, cs, p->ev_tau, &hook);
    if (rc != PPL_OK) return rc;
    PPL_CUDA(cudaStreamSynchronize(st[0]));
    PPL_CUDA(cudaStreamSynchronize(st[1]));
    PPL_CUDA(cudaStreamSynchronize(cs));
    const uint64_t nT = (uint64_t)rows * row_bytes;
    if (h2d) *h2d = (uint64_t)nL + 2 * nT;
    if (d2h) *d2h = nT;
    rc = pplapi::verify_harvest(p, nullptr);
    // (synchronous mode 2 harvested L's word at the head of the call; the chunk checks have set t2's word since)
    if (rc == PPL_OK && p->verify && p->vflags_host[1]) rc = fail(PPL_ERR_PRECONDITION);
    return rc;
}

// An error half way leaves copies and kernels in flight on three streams that read and write the caller's host buffers:
// wait for them before the error is returned, so that the caller may free or reuse its buffers.
static int apply_host_full(ppl_plan_s *p, const double *Lh, const double *t2h, double *Rh, uint64_t *h2d, uint64_t *d2h) {
    const int rc = apply_host_full_queue(p, Lh, t2h, Rh, h2d, d2h);
    if (rc != PPL_OK) {
        for (cudaStream_t st : {p->gen, p->hs2, p->host_stream})
            if (st && cudaStreamSynchronize(st) != cudaSuccess) (void)cudaGetLastError();
        p->verify_pending = 0;
    }
    return rc;
}


// ------------------------------------------------------------------------------------------------------------------
// PPL_SYM_NONE / PPL_SYM_PAIR on host operands (even nvirt, TMA kernels): nothing is assumed of L, and in PPL_SYM_NONE
// nothing of t2 -- the setting of the paper's own benchmark (unstructured random arrays).
//
// Every W tile (A, B) contracts with ALL of t2, so t2 is copied whole and stays resident.  L is read as two row panels
// per tile, L[:, A, :] and L[:, B, :] (each nchol rows of |A| nvirt contiguous doubles: a 2-D copy), so it need not be
// resident: panel A is kept for the whole row of tiles (two buffers: row k + 1 arrives while row k computes), panel B
// rides a ring with one buffer per W slot.  In PPL_SYM_NONE the tiles of row A are the only writers of R[:, :, A, :]:
// that slab ([nocc^2][|A| nvirt], again a 2-D copy) travels in before the row's first reduction and out behind its last,
// double-buffered, on copy streams of their own.  In PPL_SYM_PAIR the mirror image R[j,i,b,a] of every tile lands in
// the slab of its b-block, so R stays resident and travels whole.  The paper moves its chunks in sequence (H2D, two
// tensordots, D2H per chunk: PAPER.md:146-181); here the copy engines run beside the GEMMs the whole time.
//
// Streams: `in` all H2D copies in program order; `gen` step 0 (the plan's producer stream); `cs` step 1 + reduction;
// `out` the D2H copies.  Events guard every buffer in both directions (filled -> may be read, read -> may be refilled).
// ------------------------------------------------------------------------------------------------------------------
static int host_events(ppl_plan_s *p) {
    ppl_plan_s::HostStream &h = p->hsn;
    if (!h.events) {
        bool ok = cudaStreamCreateWithFlags(&h.in, cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaStreamCreateWithFlags(&h.out, cudaStreamNonBlocking) == cudaSuccess;
        auto ev = [&](cudaEvent_t *e) { ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess; };
        for (int i = 0; i < 2; ++i) {
            ev(&h.ev_pa[i]);
            ev(&h.ev_pafree[i]);
            ev(&h.ev_rsin[i]);
            ev(&h.ev_rsdone[i]);
            ev(&h.ev_rsfree[i]);
            ev(&h.ev_chunk[i]);
        }
        for (int i = 0; i < MAX_RING; ++i) {
            ev(&h.ev_pb[i]);
            ev(&h.ev_pbfree[i]);
        }
        ev(&h.ev_t2);
        ev(&h.ev_fork);
        if (!ok) {
            (void)cudaGetLastError();
            return fail(PPL_ERR_CUDA);
        }
        h.events = true;
    }
    return PPL_OK;
}

static int host_tiles_setup(ppl_plan_s *p, bool panels, bool slabs) {
    ppl_plan_s::HostStream &h = p->hsn;
    const size_t nT = (size_t)p->o * p->o * p->vv * 8, nL = (size_t)p->x * p->vv * 8;
    int rc = host_events(p);
    if (rc != PPL_OK) return rc;
    bool ok = dev_alloc(&p->dT, nT);
    if (ok && !slabs) ok = dev_alloc(&p->dR, nT);
    if (ok && slabs) {
        const size_t slab = (size_t)p->o * p->o * p->T * p->v * 8;
        if (h.slab_bytes < slab) {  // (the PPL_SYM_FULL route sizes the same two buffers for its own slabs)
            for (int i = 0; i < 2; ++i) dev_free(&h.rs[i]);
            h.slab_bytes = slab;
        }
        for (int i = 0; i < 2 && ok; ++i) ok = dev_alloc(&h.rs[i], h.slab_bytes);
        if (!ok) h.slab_bytes = 0;
    }
    if (ok && panels) {
        h.panel_bytes = (size_t)p->x * p->T * p->v * 8;
        h.npb = p->ring;
        for (int i = 0; i < 2 && ok; ++i) ok = dev_alloc(&h.pa[i], h.panel_bytes);
        for (int i = 0; i < h.npb && ok; ++i) ok = dev_alloc(&h.pb[i], h.panel_bytes);
    }
    if (ok && !panels) ok = dev_alloc(&p->dL, nL);
    return ok ? PPL_OK : fail(PPL_ERR_ALLOC);
}

static int apply_host_tiles_queue(ppl_plan_s *p, const double *Lh, const double *t2h, double *Rh, bool panels, uint64_t *h2d,
                                  uint64_t *d2h) {
    ppl_plan_s::HostStream &h = p->hsn;
    const bool slabs = p->sym == PPL_SYM_NONE;
    int rc = host_tiles_setup(p, panels, slabs);
    if (rc != PPL_OK) return rc;
    const int v = p->v, o2 = p->o * p->o, ntiles = (int)p->tiles.size();
    const size_t nT = (size_t)o2 * p->vv * 8, nL = (size_t)p->x * p->vv * 8, vrow = (size_t)p->vv * 8;
    cudaStream_t cs = p->host_stream, gen = p->gen, in = h.in, out = h.out;
    uint64_t up = 0, down = 0;
    // panel of the a's [a0, a0 + ta): nchol rows of ta * nvirt doubles, row pitch nvirt^2 on the host, dense on the device
    auto panel_in = [&](double *dst, int a0, int ta) -> int {
        PPL_CUDA(cudaMemcpy2DAsync(dst, (size_t)ta * v * 8, Lh + (size_t)a0 * v, vrow, (size_t)ta * v * 8, (size_t)p->x,
                                   cudaMemcpyHostToDevice, in));
        up += (uint64_t)ta * v * 8 * p->x;
        return PPL_OK;
    };
    CUtensorMap mapL, mapT;
    if (!panels) {
        PPL_CUDA(cudaMemcpyAsync(p->dL, Lh, nL, cudaMemcpyHostToDevice, in));
        up += nL;
        PPL_CUDA(cudaEventRecord(h.ev_pa[0], in));
        if (pplapi::map_2d(&mapL, p->dL, (uint64_t)p->vv, (uint64_t)p->x, vrow, 16, ppl::BK) != PPL_OK) return fail(PPL_ERR_CUDA);
    }
    if (pplapi::map_2d(&mapT, p->dT, (uint64_t)p->vv, (uint64_t)o2, vrow, ppl::BK, pplapi::step1_box_rows(p)) != PPL_OK)
        return fail(PPL_ERR_CUDA);
    bool t2_queued = false;
    auto t2_in = [&]() -> int {  // behind the operands of the first step 0: step 1 is the first kernel that needs t2
        if (t2_queued) return PPL_OK;
        t2_queued = true;
        PPL_CUDA(cudaMemcpyAsync(p->dT, t2h, nT, cudaMemcpyHostToDevice, in));
        up += nT;
        if (!slabs) {
            PPL_CUDA(cudaMemcpyAsync(p->dR, Rh, nT, cudaMemcpyHostToDevice, in));
            up += nT;
        }
        PPL_CUDA(cudaEventRecord(h.ev_t2, in));
        return PPL_OK;
    };
    int row = -1;  // index of the current row of tiles (tiles are a-block major: ppl_plan.cpp, build_tiles)
    int nb_copy = 0;  // B panels copied so far (ring position)
    for (int k = 0; k < ntiles; ++k) {
        const Tile &t = p->tiles[k];
        const bool first = k == 0 || p->tiles[k - 1].a0 != t.a0, last = k + 1 == ntiles || p->tiles[k + 1].a0 != t.a0;
        if (first) ++row;
        const int ra = row & 1, slot = k % p->ring;
        const bool diag = t.b0 == t.a0;
        int pbs = -1;
        // ---- copies in ----
        if (first && panels) {
            if (row >= 2) PPL_CUDA(cudaStreamWaitEvent(in, h.ev_pafree[ra], 0));
            if ((rc = panel_in(h.pa[ra], t.a0, t.ta)) != PPL_OK) return rc;
            PPL_CUDA(cudaEventRecord(h.ev_pa[ra], in));
        }
        if (panels && !diag) {
            pbs = nb_copy % h.npb;
            if (nb_copy >= h.npb) PPL_CUDA(cudaStreamWaitEvent(in, h.ev_pbfree[pbs], 0));
            if ((rc = panel_in(h.pb[pbs], t.b0, t.tb)) != PPL_OK) return rc;
            PPL_CUDA(cudaEventRecord(h.ev_pb[pbs], in));
            ++nb_copy;
        }
        if ((rc = t2_in()) != PPL_OK) return rc;
        if (first && slabs) {
            if (row >= 2) PPL_CUDA(cudaStreamWaitEvent(in, h.ev_rsfree[ra], 0));
            PPL_CUDA(cudaMemcpy2DAsync(h.rs[ra], (size_t)t.ta * v * 8, Rh + (size_t)t.a0 * v, vrow, (size_t)t.ta * v * 8, (size_t)o2,
                                       cudaMemcpyHostToDevice, in));
            up += (uint64_t)t.ta * v * 8 * o2;
            PPL_CUDA(cudaEventRecord(h.ev_rsin[ra], in));
        }
        // ---- producer: step 0 ----
        if (k >= p->ring) PPL_CUDA(cudaStreamWaitEvent(gen, p->ev_free[slot], 0));
        CUtensorMap mA, mB;
        if (panels) {
            if (first) PPL_CUDA(cudaStreamWaitEvent(gen, h.ev_pa[ra], 0));
            if (pplapi::map_2d(&mA, h.pa[ra], (uint64_t)t.ta * v, (uint64_t)p->x, (size_t)t.ta * v * 8, 16, ppl::BK) != PPL_OK)
                return fail(PPL_ERR_CUDA);
            if (!diag) {
                PPL_CUDA(cudaStreamWaitEvent(gen, h.ev_pb[pbs], 0));
                if (pplapi::map_2d(&mB, h.pb[pbs], (uint64_t)t.tb * v, (uint64_t)p->x, (size_t)t.tb * v * 8, 16, ppl::BK) != PPL_OK)
                    return fail(PPL_ERR_CUDA);
            }
            rc = pplapi::step0_tile(p, t, &mA, 0, diag ? &mA : &mB, 0, p->slot[slot], gen);
        } else {
            if (k == 0) PPL_CUDA(cudaStreamWaitEvent(gen, h.ev_pa[0], 0));
            rc = pplapi::step0_tile(p, t, &mapL, t.a0 * v, &mapL, t.b0 * v, p->slot[slot], gen);
        }
        if (rc != PPL_OK) return rc;
        if (panels && !diag) PPL_CUDA(cudaEventRecord(h.ev_pbfree[pbs], gen));
        if (panels && last) PPL_CUDA(cudaEventRecord(h.ev_pafree[ra], gen));
        PPL_CUDA(cudaEventRecord(p->ev_ready[slot], gen));
        // ---- consumer: step 1, reduction ----
        PPL_CUDA(cudaStreamWaitEvent(cs, p->ev_ready[slot], 0));
        if (k == 0) {
            PPL_CUDA(cudaStreamWaitEvent(cs, h.ev_t2, 0));
            // PPL_SYM_PAIR relies on pair-symmetric t2: verified on the resident copy (PPL_OPT_VERIFY_INPUTS; L: no precondition)
            if (p->sym != PPL_SYM_NONE && p->verify && (rc = pplapi::verify_begin(p, nullptr, p->dT, PPL_LAYOUT_IJAB, cs)) != PPL_OK)
                return rc;
        }
        if ((rc = pplapi::step1_tile(p, &mapT, p->dT, slot, t, cs)) != PPL_OK) return rc;
        PPL_CUDA(cudaEventRecord(p->ev_free[slot], cs));
        if (slabs) {
            if (first) PPL_CUDA(cudaStreamWaitEvent(cs, h.ev_rsin[ra], 0));
            // the slab holds R[i][j][a - a0][b]: strides (o ta v, ta v, v, 1) from the address element (0,0,0,0) would have
            const int64_t tav = (int64_t)t.ta * v;
            rc = pplapi::reduce_tile(p, t, h.rs[ra], (int64_t)p->o * tav, tav, v, 1, 1.0, 1.0, cs, (int64_t)t.a0 * v);
        } else {
            rc = pplapi::reduce_tile(p, t, p->dR, (int64_t)p->o * p->vv, p->vv, v, 1, 1.0, 1.0, cs);
        }
        if (rc != PPL_OK) return rc;
        if (slabs && last) {  // the row is complete: its slab travels out
            PPL_CUDA(cudaEventRecord(h.ev_rsdone[ra], cs));
            PPL_CUDA(cudaStreamWaitEvent(out, h.ev_rsdone[ra], 0));
            PPL_CUDA(cudaMemcpy2DAsync(Rh + (size_t)t.a0 * v, vrow, h.rs[ra], (size_t)t.ta * v * 8, (size_t)t.ta * v * 8, (size_t)o2,
                                       cudaMemcpyDeviceToHost, out));
            down += (uint64_t)t.ta * v * 8 * o2;
            PPL_CUDA(cudaEventRecord(h.ev_rsfree[ra], out));
        }
    }
    if (!slabs) {
        PPL_CUDA(cudaMemcpyAsync(Rh, p->dR, nT, cudaMemcpyDeviceToHost, cs));
        down += nT;
    }
    for (cudaStream_t st : {in, gen, cs, out}) PPL_CUDA(cudaStreamSynchronize(st));
    if (h2d) *h2d = up;
    if (d2h) *d2h = down;
    return pplapi::verify_harvest(p, nullptr);
}

static int apply_host_tiles(ppl_plan_s *p, const double *Lh, const double *t2h, double *Rh, uint64_t *h2d, uint64_t *d2h) {
    // L whole when it fits beside t2 (and R, when R is resident) with room to spare, as row panels otherwise
    const size_t nT = (size_t)p->o * p->o * p->vv * 8, nL = (size_t)p->x * p->vv * 8;
    bool panels = p->dbg.host_panels == 1;
    if (p->dbg.host_panels == 0 && !p->dL) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) {
            (void)cudaGetLastError();
            return fail(PPL_ERR_CUDA);
        }
        size_t need = nL + ((size_t)2 << 30);
        if (!p->dT) need += nT;
        if (p->sym != PPL_SYM_NONE && !p->dR) need += nT;
        panels = need > free_b;
    }
    int rc = apply_host_tiles_queue(p, Lh, t2h, Rh, panels, h2d, d2h);
    if (rc != PPL_OK) {
        for (cudaStream_t st : {p->hsn.in, p->gen, p->host_stream, p->hsn.out})
            if (st && cudaStreamSynchronize(st) != cudaSuccess) (void)cudaGetLastError();
        p->verify_pending = 0;
        p->vq_n = 0;
        if (rc == PPL_ERR_ALLOC) {  // leave nothing half-allocated behind: a later call may take another route
            for (int i = 0; i < 2; ++i) {
                dev_free(&p->hsn.pa[i]);
                dev_free(&p->hsn.rs[i]);
            }
            p->hsn.slab_bytes = 0;
            for (int i = 0; i < MAX_RING; ++i) dev_free(&p->hsn.pb[i]);
        }
    }
    return rc;
}

extern "C" {

int ppl_apply_host(ppl_plan_t *p, const double *Lh, const double *t2h, double *Rh, uint64_t *h2d, uint64_t *d2h) {
    int cur = -1;
    if (!p || !Lh || !t2h || !Rh) return fail(PPL_ERR_INVALID_ARG);
    if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device) {  // the plan's buffers and streams live on its own device
        (void)cudaGetLastError();
        return fail(PPL_ERR_INVALID_ARG);
    }
    const bool aligned = (((uintptr_t)Lh | (uintptr_t)t2h | (uintptr_t)Rh) & 7) == 0;
    if (p->sym == PPL_SYM_FULL && p->full_ok && aligned) return apply_host_full(p, Lh, t2h, Rh, h2d, d2h);
    if ((p->sym == PPL_SYM_NONE || p->sym == PPL_SYM_PAIR) && p->use_tma && p->vec16 && aligned && !p->small_ok)
        return apply_host_tiles(p, Lh, t2h, Rh, h2d, d2h);
    const size_t nL = (size_t)p->x * p->v * p->v * 8, nT = (size_t)p->o * p->o * p->v * p->v * 8;
    if (!dev_alloc(&p->dL, nL)) return fail(PPL_ERR_ALLOC);
    if (!dev_alloc(&p->dT, nT) || !dev_alloc(&p->dR, nT)) {
        dev_free(&p->dT);
        dev_free(&p->dR);
        return fail(PPL_ERR_ALLOC);
    }
    cudaStream_t s = p->host_stream;
    PPL_CUDA(cudaMemcpyAsync(p->dL, Lh, nL, cudaMemcpyHostToDevice, s));
    PPL_CUDA(cudaMemcpyAsync(p->dT, t2h, nT, cudaMemcpyHostToDevice, s));
    PPL_CUDA(cudaMemcpyAsync(p->dR, Rh, nT, cudaMemcpyHostToDevice, s));
    int rc = ppl_apply(p, p->dL, p->dT, p->dR, s);
    if (rc != PPL_OK && cudaStreamSynchronize(s) != cudaSuccess) (void)cudaGetLastError();  // the queued H2D copies read the caller's buffers
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
    if (rc == PPL_OK) rc = pplapi::verify_harvest(p, nullptr);  // the call has synchronised: report a violated precondition at once
    return rc;
}

}  // extern "C"
