// ppl_plan.h -- internal: the plan object and the host planner's interface.  Plain C++ (CUDA headers are used for
// TYPES only -- streams, events, tensor maps -- so ppl_plan.cpp compiles and links with g++ alone, no nvcc, no CUDA call).
#pragma once
#include <cuda.h>           // CUtensorMap
#include <driver_types.h>   // cudaStream_t, cudaEvent_t, cudaGraphExec_t
#include <vector_types.h>   // int2

#include <cstddef>
#include <cstdint>
#include <vector>

#include "../../include/ppl.h"
#include "ppl_layout.h"

namespace pplh {

struct SplitChoice {
    int splitk = 1, k_per_split = ppl::BK;
    double seconds = 0;
};

// Row tiling of the M side of step 1.  TMA kernels: 8-row blocks dealt to 2*tiles_m half-tiles of `base` or `base+1`
// blocks (ppl::MSplit); cp.async kernels: uniform tiles of 128 rows.
struct MGeom {
    int tiles_m = 1, base = 0, rem = 0;
    int ni = 8;         // template instance (TMA box of the A operand: 16*ni rows)
    double rows = 128;  // average rows computed per CTA tile (cost model)
};

struct Tile {
    int a0, ta, b0, tb;
    int mirror;
    SplitChoice full;    // step 1 over K = nvirt^2                (PPL_SYM_NONE / PPL_SYM_PAIR)
    SplitChoice sp, sm;  // step 1 over the packed K+ / K- ranges  (PPL_SYM_PAIR_SA)
};

// PPL_SYM_FULL: one tile = (a-block A of 16) x (a group of b's), one slab = all tiles of one A
struct FullTile {
    int A0, ta;      // a-block
    int bg0, nb;     // first b of the group, number of b's in it
    int tbp;         // nb rounded up to a multiple of 16: W-tile rows are a_l*tbp + b_l
    int k0p, k0m;    // first packed (c<=d) / (c<d) index with c >= A0: start of the use-1 contraction range
    int k1p, k1m;    // first packed index with c >= A0+16: start of the use-2 output range
    SplitChoice sp, sm;
    // memory-tight mode: step 0 runs per tile on the full (b in group, d >= A0) rectangle into a strip of the tile's rows
    size_t chunk_off = 0;
    int tiles_n = 0;
    // range tiles (the default outside the memory-tight form): the W+- rows are a run of the packed pair index of (a <= b),
    // a in the slab -- no zero rows for a > b and no rounding of the b count, only the holes of the packed layout
    int range = 0;
    int kp0 = 0, np = 0, npr = 0;  // plus: first packed index, rows, rows rounded up to 16 (the k-tiles of use 2)
    int km0 = 0, nm = 0, nmr = 0;  // minus rows of the same pairs
    int nzm = 0, zrows_m[24] = {};  // minus rows no pair writes (holes, tail): zeroed by the fold
};
struct FullSlab {
    int A0, ta;
    int tiles_m, tiles_n;  // step-0 CTA tiles: 128 rows (c, a_l), 128 columns (8 chunks of 16 d's)
    size_t chunk_off;      // first entry of this slab in the chunk table
    int tile_begin, tile_end;
    double flops0;
};

constexpr int MAX_RING = 4;
constexpr double PEAK_FLOPS = 37.2e12;  // nominal FP64 (148 SM x 64 FMA/clk x 2 x 1.965 GHz); planner cost model only
constexpr double HBM_BPS = 6.0e12;      // planner cost model only
constexpr double GRAPH_AUTO_FLOPS = 5.0e9;   // ppl_plan_set_graph(-1): measured -- tiny 47.7 -> 37.9 us, small (1.7e9) 270 -> 231 us with the graph; (10,100,400) (2.8e10) 1.44 -> 1.51 ms, medium 26.1 -> 26.8 ms without
constexpr double LAUNCH_S = 4e-6;

inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

}  // namespace pplh

struct ppl_plan_s {
    int o = 0, v = 0, x = 0;
    int sym = PPL_SYM_PAIR_SA;
    int sa_ok = 0;        // the workspace holds the packed operands of PPL_SYM_PAIR_SA
    int T = 0;            // tile edge (ta = tb = T except at the ragged edge)
    int nblk = 0;
    int ring = 1;
    int vec16 = 0;
    int num_sms = 148;
    int device = -1;      // the CUDA device ppl_plan ran on: workspace, streams and events live there (-1: ppl_plan_dry)
    int use_tma = 0;      // 1: persistent TMA/mbarrier kernels; 0: cp.async kernels
    int64_t vv = 0;       // nvirt^2 = row length of an un-packed W tile / of t2
    int vp = 0;           // nvirt rounded up to even: the geometry of every PACKED operand (tau+-, W+-, R+-acc) and of the
    int64_t vvp = 0;      // whole PPL_SYM_FULL path; for odd nvirt the pad index carries exact zeros
    double *Lpad = nullptr;  // PPL_SYM_FULL with odd nvirt: L copied into [x][vp][vp] (TMA needs 16-byte rows), inside fws
    // packed geometry (PPL_SYM_PAIR_SA)
    int Mp = 0, Mm = 0;   // rows (i<=j), (i<j)
    int Kp = 0, Km = 0;   // extents of the packed column indices of (c<=d), (c<d), holes included
    int KpT = 0, KmT = 0; // number of pairs (c<=d), (c<d)
    int64_t ldp = 0, ldm = 0;
    int bm_full = 128, bm_p = 128, bm_m = 128;  // step-1 CTA tile rows (TMA box: 16*NI)
    pplh::MGeom mg_full, mg_p, mg_m;                  // row tiling of nocc^2 / the packed (i<=j) / (i<j) rows
    size_t cap = 0;
    size_t x_bytes = 0, slot_bytes = 0, part_bytes = 0, tau_bytes = 0, ws_bytes = 0;
    unsigned char *ws = nullptr;
    double *X = nullptr;                   // SA: step-0 output tile [T*T][vv], folded into a ring slot
    double *slot[pplh::MAX_RING] = {nullptr, nullptr, nullptr, nullptr};  // W tile, or W+ [T*T][ldp] followed by W- [T*T][ldm]
    double *part = nullptr;
    double *taup = nullptr, *taum = nullptr;
    double *tperm = nullptr;               // un-packed modes with PPL_LAYOUT_IAJB input: t2 permuted (lazy)
    int *vflags_host = nullptr;            // [32] mapped pinned host words written by k_check_inputs: [0..1] the per-apply verification
                                           // (PPL_OPT_VERIFY_INPUTS), [2..3] ppl_check_inputs
    cudaEvent_t ev_verify = nullptr;
    int verify = 1;                        // PPL_OPT_VERIFY_INPUTS
    int verify_pending = 0;                // 1: a k_check_inputs launch is outstanding (ev_verify follows it)
    // the check CTAs of k_small_fused (launch-bound shapes): up to two applies outstanding, oldest first.  Apply number `seq`
    // uses slot seq & 1: flags in vflags_host[8 + 8 slot + 0..1], its sequence number arrives in vflags_host[8 + 8 slot + 4]
    int *vdone_dev = nullptr;              // [2] device counters of finished check CTAs, one per slot
    int vseq = 0;                          // sequence number of the last fused check
    int vq_seq[2] = {0, 0}, vq_n = 0;      // outstanding sequence numbers
    cudaEvent_t ev_vq[2] = {nullptr, nullptr};  // one per slot, recorded right behind the fused launch on ITS stream: what the
                                           // harvest asks when the sequence number is slow to arrive (the caller's streams are
                                           // borrowed and may differ between applies or be destroyed; an event stays valid)
    std::vector<pplh::Tile> tiles;
    cudaStream_t gen = nullptr, host_stream = nullptr;
    cudaEvent_t ev_in = nullptr, ev_ready[pplh::MAX_RING] = {}, ev_free[pplh::MAX_RING] = {};
    double *dL = nullptr, *dT = nullptr, *dR = nullptr;  // ppl_apply_host staging
    double *hstage[2] = {nullptr, nullptr};              // ppl_apply_host in PPL_SYM_FULL: two chunk buffers for t2 / R
    int hchunk_rows = 0;                                 // (i,j) rows per chunk
    cudaStream_t hs2 = nullptr;                          // second chunk stream of ppl_apply_host (the first is `gen`)
    cudaEvent_t ev_tau = nullptr, ev_done = nullptr;     // tau+- complete / all slabs done
    // ppl_apply_host in the un-packed modes (ppl_host.cu): L row panels, R slabs, their streams and events
    struct HostStream {
        double *pa[2] = {nullptr, nullptr};              // panel L[:, A, :] of the current / next row of tiles: [x][ta * v]
        double *pb[pplh::MAX_RING] = {};                 // panels L[:, B, :], one per W slot
        double *rs[2] = {nullptr, nullptr};              // R slab [o*o][ta * v] of the current / next row (PPL_SYM_NONE)
        size_t panel_bytes = 0, slab_bytes = 0;
        int npb = 0;
        cudaStream_t in = nullptr, out = nullptr;        // H2D copies / D2H copies
        cudaEvent_t ev_pa[2] = {}, ev_pafree[2] = {}, ev_pb[pplh::MAX_RING] = {}, ev_pbfree[pplh::MAX_RING] = {};
        cudaEvent_t ev_rsin[2] = {}, ev_rsdone[2] = {}, ev_rsfree[2] = {}, ev_t2 = nullptr, ev_fork = nullptr;
        cudaEvent_t ev_chunk[2] = {};                    // PPL_SYM_FULL: chunk k of t2 is packed (recorded on chunk stream k & 1)
        bool events = false;
    } hsn;
    double f_step0 = 0, f_step1 = 0;
    CUtensorMap mapW[pplh::MAX_RING], mapWp[pplh::MAX_RING], mapWm[pplh::MAX_RING], mapTp, mapTm;  // plan-owned operands
    // ---- PPL_SYM_FULL (own allocation `fws`; shares taup/taum with PPL_SYM_PAIR_SA) ----
    int full_ok = 0;
    int full_tight = 0;                        // 1: the strip holds one (slab; b-group) tile, step 0 runs per tile without the b<->d image
    int tbg = 0;                               // b-group width (multiple of 16)
    size_t fws_bytes = 0;
    unsigned char *fws = nullptr;
    double *fX = nullptr;                      // strip [16*v rows (a_l*v + b)][vv]
    double *fX2 = nullptr;                     // second strip (when it fits): step 0 of slab k+1 runs on `fs0` while slab k is folded
    cudaStream_t fs0 = nullptr;                // producer stream of step 0 (two strips only)
    cudaEvent_t ev_fork = nullptr, ev_s0[2] = {nullptr, nullptr}, ev_xfree[2] = {nullptr, nullptr};
    int fslots = 1;                            // W+- slots (2 when they fit: the fold of tile k+1 overlaps the GEMMs of tile k)
    double *fWp[2] = {nullptr, nullptr}, *fWm[2] = {nullptr, nullptr};  // W+- tile [16*tbg][ldp], [16*tbg][ldm]
    double *fpart = nullptr;
    double *raccp = nullptr, *raccm = nullptr; // R+- accumulators [Mp][ldp], [Mm][ldm]
    int2 *fchunks = nullptr;
    double *Lq = nullptr;                      // packed diagonal 16 x 16 blocks of L: [x][ldq] (ppl_kernels_full.cuh, k_pack_diag)
    int nfull = 0;                             // full 16-blocks of the (padded) virtual index
    int64_t ldq = 0;
    int diag_pack = 0;
    CUtensorMap mapLq;
    ppl_debug_opts_t dbg = {};
    // what full_plan (host) sized for full_allocate (device)
    int full_planned = 0;
    size_t fx_bytes = 0, lq_bytes = 0, lpad_bytes = 0;
    bool two_strips = false;
    std::vector<int2> chunks_host;             // chunk table of step 0 (copied to fchunks)
    size_t fpart_bytes = 0;
    size_t fpart_m_off = 0;                    // doubles: the minus partials start here (fixed: + and - run on different streams)
    std::vector<pplh::FullSlab> slabs;
    std::vector<pplh::FullTile> ftiles;
    double ff_step0 = 0, ff_step1 = 0;
    cudaStream_t fs[4] = {nullptr, nullptr, nullptr, nullptr};  // side streams of the four step-1 GEMMs of a tile
    cudaEvent_t ev_fold[2] = {nullptr, nullptr}, evg[2][4] = {};
    CUtensorMap mapFWp[2], mapFWm[2], mapFWpT[2], mapFWmT[2];  // the W+- tile as the B operand of use 1 (box 16 x 128 rows) / use 2 (box 16 x 16 rows)
    // ---- CUDA graph of one apply (launch-bound shapes; ppl_plan_set_graph) ----
    // ---- the one-kernel path of launch-bound shapes (ppl_kernels_small.cuh) ----
    int small_ok = 0;                          // ppl_apply takes it (whatever the symmetry mode; pair symmetry is used when the mode allows)
    double fs_step0[2] = {0, 0}, fs_step1[2] = {0, 0};  // its executed flops without / with pair symmetry
    int small_items[2] = {0, 0};
    double *small_Lp = nullptr, *small_tp = nullptr;  // copies with even-length rows for its bulk copies (odd nvirt, 'iajb' t2, misaligned buffers)
    int dry = 0;                               // ppl_plan_dry: geometry only, the plan owns nothing on the device
    int graph_mode = -1;                       // -1: auto (graph when the executed flops are below GRAPH_AUTO_FLOPS), 0: off, 1: on
    cudaStream_t gcap = nullptr;               // capture origin (never the caller's stream: the legacy stream cannot capture)
    cudaGraphExec_t gexec = nullptr;           // the instantiated apply for the key below
    struct GraphKey {
        const double *L = nullptr, *t2 = nullptr;
        double *R = nullptr;
        ppl_opts_t opts = {0, 0, 0.0, 0.0};
        int sym = -1;
    } gkey;
};


namespace pplh {

int fail(int code);  // records the code for ppl_last_error() and returns it
int fail_peek();
MGeom m_geom_tma(int M, int nmax);
MGeom m_geom_plain(int M);
SplitChoice choose_split(int M, int N, int64_t K, int sms, const MGeom &mg, size_t part_cap = ~(size_t)0);
int build_tiles(ppl_plan_s *p);
int full_plan(ppl_plan_s *p, size_t room);
ppl_plan_s *plan_host(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t cap, int num_sms, bool use_tma,
                      const ppl_debug_opts_t *dbg, int *rc_out);
bool dims_ok(int nocc, int nvirt, int nchol);
int full_min_v(const ppl_plan_s *p);
bool graph_wanted(const ppl_plan_s *p);
constexpr int SMALL_SW_HOST = 4;  // b's per work item of the one-kernel path (= ppl::SMALL_SW)

}  // namespace pplh
