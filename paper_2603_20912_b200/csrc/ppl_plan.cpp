// ppl_plan.cpp -- the host planner of libppl: everything that follows from (nocc, nvirt, nchol), a byte
// budget and an SM count -- packed geometry, row tiling of step 1, tile edge, ring depth, split-K, the slabs / tiles / chunk
// table of PPL_SYM_FULL, buffer sizes, flop accounting.  Plain C++: no CUDA call, compiles and links with g++ alone
// (tests/test_planner_cpu.py builds it that way), which is what ppl_plan_dry runs on a machine without a GPU.
#include "ppl_plan.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

namespace pplh {

namespace {
thread_local int g_last_error = PPL_OK;
inline int2 make_int2(int x, int y) {
    int2 r;
    r.x = x;
    r.y = y;
    return r;
}
}  // namespace
int fail(int code) {
    g_last_error = code;
    return code;
}
int fail_peek() { return g_last_error; }

// ------------------------------------------------------------------------------------------
// Planner: the analogue of the paper's memory functions (Table 1) -- but what
// is being sized is the W-tile ring in HBM, not host->device batches.  For a candidate tile edge
// T it estimates the time of one apply from CTA-wave counts of both GEMMs (CTA tile 128x128x16 on
// `sms` SMs), the best split-K per tile shape, and the streaming traffic.
// ------------------------------------------------------------------------------------------

// TMA kernels: the fewest CTA tiles of at most 16*10 rows, rows dealt in 8-row blocks as evenly as possible
// (ppl_kernels_tma.cuh, MSplit): padding < 8 rows in all.  nmax: largest template instance to use (debug override).
// Every warp row gets ni or ni - 1 blocks: the only two cases the kernels are compiled for.
MGeom m_geom_tma(int M, int nmax) {
    MGeom g;
    const int blocks = (std::max(M, 1) + 7) / 8;
    g.tiles_m = (blocks + 2 * nmax - 1) / (2 * nmax);
    g.base = blocks / (2 * g.tiles_m);
    g.rem = blocks % (2 * g.tiles_m);
    g.ni = g.base + (g.rem > 0 ? 1 : 0);  // 1 .. nmax
    g.rows = 8.0 * blocks / g.tiles_m;
    return g;
}
MGeom m_geom_plain(int M) {
    MGeom g;
    g.tiles_m = (std::max(M, 1) + ppl::BM - 1) / ppl::BM;
    return g;
}

SplitChoice choose_split(int M, int N, int64_t K, int sms, const MGeom &mg, size_t part_cap) {
    SplitChoice best;
    if (M <= 0 || N <= 0 || K <= 0) return best;
    const int tiles = mg.tiles_m * ((N + ppl::BN - 1) / ppl::BN);
    const int nkt = (int)((K + ppl::BK - 1) / ppl::BK);
    const double tau = 2.0 * mg.rows * ppl::BN * ppl::BK / (PEAK_FLOPS / sms);  // one k-tile on one SM
    best = SplitChoice{1, nkt * ppl::BK, 1e300};
    const int smax = std::max(1, std::min(nkt / 8 + 1, 64));
    for (int s = 1; s <= smax; ++s) {
        const int kt_per = (nkt + s - 1) / s;
        const int s_eff = (nkt + kt_per - 1) / kt_per;  // no empty splits
        if (s_eff != s) continue;
        if ((size_t)s * M * N * 8 > part_cap && s > 1) continue;
        const double waves = std::ceil((double)tiles * s / sms);
        const double t = waves * (kt_per + 6) * tau                      // +6: pipeline fill / epilogue
                         + (double)(s + 2) * M * N * 8.0 / HBM_BPS;      // partials written + read by the reduce
        if (t < best.seconds) best = SplitChoice{s, kt_per * ppl::BK, t};
    }
    return best;
}

double step0_seconds(int ta, int tb, int v, int x, int sms) {
    // (64-bit: with nvirt >= 2431 a whole-range tile edge has more than 2^31 CTA tiles -- found by UBSan, tests/test_planner_sanitizers_cpu.py)
    const int64_t tiles = (((int64_t)ta * v + ppl::BM - 1) / ppl::BM) * (((int64_t)tb * v + ppl::BN - 1) / ppl::BN);
    const int nkt = (x + ppl::BK - 1) / ppl::BK;
    const double tau = 2.0 * ppl::BM * ppl::BN * ppl::BK / (PEAK_FLOPS / sms);
    return std::ceil((double)tiles / sms) * (nkt + 6) * tau;
}

struct Geometry {  // what depends on (o, v) only
    int64_t vv;
    int M, Mp, Mm, Kp, Km;
    int64_t ldp, ldm;
    MGeom mg_full, mg_p, mg_m;
};

struct PlanEval {
    double seconds = 1e300;
    size_t x_bytes = 0, slot_bytes = 0, part_bytes = 0;
};

// estimated seconds of one apply with tile edge T in PPL_SYM_PAIR_SA (sa = true) or PPL_SYM_PAIR
PlanEval evaluate(const Geometry &g, int o, int v, int x, int T, bool sa, int sms) {
    PlanEval ev;
    const int nblk = (v + T - 1) / T;
    const int r = v - (nblk - 1) * T;  // ragged edge
    double total = 0;
    size_t part_max = 0;
    auto count = [&](bool a_edge, bool b_edge) -> int64_t {  // executed tiles (a-block <= b-block) per shape
        if (a_edge && b_edge) return 1;
        if (a_edge && !b_edge) return 0;
        if (!a_edge && b_edge) return nblk - 1;
        return (int64_t)(nblk - 1) * nblk / 2;
    };
    for (int ae = 0; ae < 2; ++ae)
        for (int be = 0; be < 2; ++be) {
            const int64_t cnt = count(ae, be);
            if (cnt == 0) continue;
            const int ta = ae ? r : T, tb = be ? r : T;
            const int N = ta * tb;
            const SplitChoice full = choose_split(g.M, N, g.vv, sms, g.mg_full);
            size_t part = (size_t)full.splitk * g.M * N * 8;
            double compute, dram;
            if (sa) {
                const SplitChoice sp = choose_split(g.Mp, N, g.Kp, sms, g.mg_p), sm = choose_split(g.Mm, N, g.Km, sms, g.mg_m);
                const double fold = 2.0 * N * g.vv * 8.0 / HBM_BPS + LAUNCH_S;
                compute = step0_seconds(ta, tb, v, x, sms) + fold + sp.seconds + sm.seconds;
                dram = (((double)g.Mp * g.ldp + (double)g.Mm * g.ldm) * 8.0 + 4.0 * N * g.vv * 8.0) / HBM_BPS;
                part = std::max(part, ((size_t)sp.splitk * g.Mp + (size_t)sm.splitk * g.Mm) * N * 8);
                total += cnt * (std::max(compute, dram) + 5 * LAUNCH_S);
            } else {
                compute = step0_seconds(ta, tb, v, x, sms) + full.seconds;
                dram = ((double)g.M * g.vv * 8.0 + 2.0 * N * g.vv * 8.0) / HBM_BPS;
                total += cnt * (std::max(compute, dram) + 3 * LAUNCH_S);
            }
            part_max = std::max(part_max, part);
        }
    ev.seconds = total;
    ev.x_bytes = sa ? align256((size_t)T * T * g.vv * 8) : 0;
    ev.slot_bytes = align256(sa ? (size_t)T * T * (g.ldp + g.ldm) * 8 : (size_t)T * T * g.vv * 8);
    ev.part_bytes = align256(part_max);
    return ev;
}

int build_tiles(ppl_plan_s *p) {
    p->tiles.clear();
    p->f_step0 = p->f_step1 = 0;
    const int T = p->T, v = p->v, M = p->o * p->o;
    const bool pair = p->sym != PPL_SYM_NONE, sa = p->sym == PPL_SYM_PAIR_SA;
    for (int ab = 0; ab < p->nblk; ++ab)
        for (int bb = (pair ? ab : 0); bb < p->nblk; ++bb) {
            Tile t;
            t.a0 = ab * T;
            t.ta = std::min(T, v - t.a0);
            t.b0 = bb * T;
            t.tb = std::min(T, v - t.b0);
            t.mirror = (pair && ab != bb) ? 1 : 0;
            const int N = t.ta * t.tb;
            if (sa) {
                t.sp = choose_split(p->Mp, N, p->Kp, p->num_sms, p->mg_p);
                t.sm = choose_split(p->Mm, N, p->Km, p->num_sms, p->mg_m);
                if (((size_t)t.sp.splitk * p->Mp + (size_t)t.sm.splitk * p->Mm) * N * 8 > p->part_bytes)
                    return PPL_ERR_WORKSPACE_TOO_SMALL;
                p->f_step1 += 2.0 * N * ((double)p->Mp * p->KpT + (double)p->Mm * p->KmT);
            } else {
                t.full = choose_split(M, N, p->vv, p->num_sms, p->mg_full, p->part_bytes);
                if ((size_t)t.full.splitk * M * N * 8 > p->part_bytes) return PPL_ERR_WORKSPACE_TOO_SMALL;
                p->f_step1 += 2.0 * M * (double)N * (double)p->vv;
            }
            p->tiles.push_back(t);
            p->f_step0 += 2.0 * p->x * (double)N * (double)p->vv;
        }
    return PPL_OK;
}

// flops of one step-1 launch as the CTA tiles execute it: rows in 8-row blocks (MSplit), columns in tiles of 128, k in tiles of 16
double gemm_flops_launched(const MGeom &mg, int M, int64_t ncols, int64_t krange) {
    if (M <= 0 || ncols <= 0 || krange <= 0) return 0;
    const double rows = 8.0 * ((M + 7) / 8);
    (void)mg;
    return 2.0 * rows * (128.0 * ((ncols + 127) / 128)) * (16.0 * ((krange + 15) / 16));
}

int full_geometry(ppl_plan_s *p, int tbg, size_t part_cap, std::vector<int2> *chunks_out, bool tight = false) {
    const int v = p->vp, TA = ppl::TA_FULL;
    p->slabs.clear();
    p->ftiles.clear();
    p->ff_step0 = p->ff_step1 = 0;
    p->fpart_bytes = 0;
    size_t part_p = 0, part_m = 0;
    std::vector<int2> chunks;
    const bool range_tiles = !tight && !p->dbg.full_rect_tiles;
    const bool diag_pack = !tight && !p->dbg.full_no_diag_pack && v >= 16;
    p->diag_pack = diag_pack ? 1 : 0;
    p->nfull = v / 16;
    p->ldq = (int64_t)std::max(p->nfull, 1) * ppl::DIAG_PACKED;
    std::vector<unsigned char> mark;
    for (int A0 = 0; A0 < v; A0 += TA) {
        FullSlab sl;
        sl.A0 = A0;
        sl.ta = std::min(TA, v - A0);
        sl.tiles_m = ((v - A0) + 7) / 8;  // 8 c's x 16 a_l per 128-row CTA tile
        sl.chunk_off = chunks.size();
        // d-block major: the 8 chunks of a CTA tile are 8 consecutive b's of one d-block, so that the b<->d image
        // X[a,d,c,b] is written as runs of 8 b's (two full 32-byte sectors, merged in L2) instead of lone doubles
        if (!tight) {
            // A ragged last d-block [dL, v) of width w < 16 would cost a whole 16-wide chunk for every b >= A0.  It is
            // covered from the other side instead: the w b's of that block against every d-block from A0 up (chunks with
            // d-block BELOW the b-block; the epilogue stores their b<->d image like that of any off-diagonal chunk), which
            // is w * ceil(r / 16) chunks instead of r (nvirt = 200, 600: w = 8, half as many).
            const int dL = A0 + (v - 1 - A0) / 16 * 16, w = v - dL;
            const bool reverse = w < 16 && (int64_t)w * ((v - A0 + 15) / 16) < (v - A0);
            // Diagonal blocks (b-block == d-block, full 16 x 16): only b <= d is needed -- 9 chunks of the packed copy Lq
            // (k_pack_diag) instead of 16 plain ones.  They go behind the plain chunks so that those keep their
            // (b even, b + 1) pairing inside the column tiles (16-byte image stores).
            for (int d0 = A0; d0 < v; d0 += 16) {
                if (reverse && d0 == dL) break;
                const bool packed = diag_pack && d0 + 16 <= v;
                for (int b = A0; b < (packed ? d0 : std::min(d0 + 16, v)); ++b) chunks.push_back(make_int2(b, d0));
            }
            if (reverse)
                for (int d0 = A0; d0 <= dL; d0 += 16)
                    for (int b = dL; b < v; ++b) chunks.push_back(make_int2(b, d0));
            if (diag_pack)
                for (int d0 = A0; d0 + 16 <= v; d0 += 16)
                    for (int j = 0; j < ppl::DIAG_PACKED / 16; ++j)
                        chunks.push_back(make_int2(-2 - d0 / 16, d0 / 16 * ppl::DIAG_PACKED + 16 * j));
            while ((chunks.size() - sl.chunk_off) % 8) chunks.push_back(make_int2(-1, 0));
        }
        sl.tiles_n = (int)((chunks.size() - sl.chunk_off) / 8);
        sl.flops0 = 2.0 * p->x * (128.0 * sl.tiles_m) * (128.0 * sl.tiles_n);
        p->ff_step0 += sl.flops0;
        sl.tile_begin = (int)p->ftiles.size();
        const int c1 = std::min(A0 + TA, v);
        // range starts are even (TMA alignment): (A0,A0) sits at an even index, and the element before
        // (A0, A0+1) in the minus triangle is a hole (A0 even)
        const int k0p = (int)ppl::kplus(A0, A0, v);
        const int k0m = A0 + 1 < v ? (int)ppl::kminus(A0, A0 + 1, v) - 1 : p->Km;
        const int k1p = c1 < v ? (int)ppl::kplus(c1, c1, v) : p->Kp;
        const int k1m = c1 + 1 < v ? (int)ppl::kminus(c1, c1 + 1, v) - 1 : p->Km;
        auto finish_tile = [&](FullTile &t, int Np, int Nm, int Kup, int Kum) {
            // Np / Nm: W+- rows contracted by use 1 (its GEMM N); Kup / Kum: W+- rows contracted by use 2 (its GEMM K)
            t.k0p = k0p;
            t.k0m = k0m;
            t.k1p = k1p;
            t.k1m = k1m;
            t.sp = choose_split(p->Mp, Np, p->Kp - t.k0p, p->num_sms, p->mg_p, part_cap / 2);
            t.sm = choose_split(p->Mm, Nm, p->Km - t.k0m, p->num_sms, p->mg_m, part_cap / 2);
            part_p = std::max(part_p, (size_t)t.sp.splitk * p->Mp * Np);
            part_m = std::max(part_m, (size_t)t.sm.splitk * p->Mm * std::max(Nm, 0));
            p->fpart_m_off = (part_p + 31) / 32 * 32;
            p->fpart_bytes = (p->fpart_m_off + part_m) * 8;
            // executed flops, as the CTA tiles run them: use 1 (contraction over J >= (A0,A0)) + use 2 (outputs J >= (A0+16,A0+16))
            p->ff_step1 += gemm_flops_launched(p->mg_p, p->Mp, Np, p->Kp - t.k0p) + gemm_flops_launched(p->mg_m, p->Mm, Nm, p->Km - t.k0m);
            p->ff_step1 += gemm_flops_launched(p->mg_p, p->Mp, p->Kp - (t.k1p & ~15), Kup) +
                           gemm_flops_launched(p->mg_m, p->Mm, p->Km - (t.k1m & ~15), Kum);
        };
        if (range_tiles) {
            // the slab's pairs (a <= b), a in the slab, are ONE run of the packed index; it is cut into tiles of at most 16 tbg
            // rows at multiples of 128 (the column tile of use 1)
            const int64_t lo = k0p, hi = ppl::kplus(A0 + sl.ta - 1, v - 1, v) + 1, Ls = hi - lo, NT = (int64_t)TA * tbg;
            const int ng = (int)((Ls + NT - 1) / NT);
            int64_t chunk = ((Ls + ng - 1) / ng + 127) / 128 * 128;
            if (chunk > NT) chunk = NT;
            int64_t prev_last_m = -1;
            for (int64_t kp0 = lo; kp0 < hi; kp0 += chunk) {
                FullTile t;
                t.A0 = A0;
                t.ta = sl.ta;
                t.bg0 = A0;
                t.nb = v - A0;
                t.tbp = 0;
                t.range = 1;
                t.kp0 = (int)kp0;
                t.np = (int)(std::min(kp0 + chunk, hi) - kp0);
                t.npr = (t.np + 15) / 16 * 16;
                // the minus rows of the tile's pairs
                int64_t first_m = -1, last_m = -1;
                int a = A0;
                for (int64_t kap = kp0; kap < kp0 + t.np; ++kap) {
                    while (a + 1 < A0 + sl.ta && ppl::kplus(a + 1, a + 1, v) <= kap) ++a;
                    const int b = a + (int)(kap - ppl::kplus(a, a, v));
                    if (b >= v || b <= a) continue;  // hole / diagonal pair
                    const int64_t km = ppl::kminus(a, b, v);
                    if (first_m < 0) first_m = km;
                    last_m = km;
                }
                if (first_m >= 0) {
                    t.km0 = (int)(first_m & ~(int64_t)1);
                    if ((int64_t)t.km0 <= prev_last_m) return PPL_ERR_INVALID_ARG;  // never: cuts fall on even indices (kplus / kminus parity = parity of b)
                    t.nm = (int)(last_m + 1 - t.km0);
                    t.nmr = (t.nm + 15) / 16 * 16;
                    prev_last_m = last_m;
                    mark.assign(t.nmr, 0);
                    a = A0;
                    for (int64_t kap = kp0; kap < kp0 + t.np; ++kap) {
                        while (a + 1 < A0 + sl.ta && ppl::kplus(a + 1, a + 1, v) <= kap) ++a;
                        const int b = a + (int)(kap - ppl::kplus(a, a, v));
                        if (b >= v || b <= a) continue;
                        mark[ppl::kminus(a, b, v) - t.km0] = 1;
                    }
                    for (int r = 0; r < t.nmr; ++r)
                        if (!mark[r]) {
                            if (t.nzm >= 24) return PPL_ERR_INVALID_ARG;  // never: <= 8 holes (one per two a's) + 15 tail rows
                            t.zrows_m[t.nzm++] = r;
                        }
                }
                finish_tile(t, t.np, t.nm, t.npr, t.nmr);
                p->ftiles.push_back(t);
            }
        } else {
            // b-groups: the 16-blocks of [A0, v) dealt into groups of at most tbg/16 blocks, as evenly as possible
            const int nblk = (v - A0 + 15) / 16, per = tbg / 16, ng = (nblk + per - 1) / per;
            int blk = 0;
            for (int gi = 0; gi < ng; ++gi) {
                const int cnt = nblk / ng + (gi < nblk % ng ? 1 : 0);
                FullTile t;
                t.A0 = A0;
                t.ta = sl.ta;
                t.bg0 = A0 + 16 * blk;
                t.nb = std::min(16 * cnt, v - t.bg0);
                t.tbp = 16 * cnt;
                blk += cnt;
                const int N = TA * t.tbp;
                finish_tile(t, N, N, N, N);
                if (tight) {  // the full (b, d) rectangle of the group: no image, twice the step-0 flops, a strip of tbp rows per a
                    t.chunk_off = chunks.size();
                    for (int d0 = A0; d0 < v; d0 += 16)
                        for (int b = t.bg0; b < t.bg0 + t.nb; ++b) chunks.push_back(make_int2(b, d0));
                    while ((chunks.size() - t.chunk_off) % 8) chunks.push_back(make_int2(-1, 0));
                    t.tiles_n = (int)((chunks.size() - t.chunk_off) / 8);
                    const double f0 = 2.0 * p->x * (128.0 * sl.tiles_m) * (128.0 * t.tiles_n);
                    sl.flops0 += f0;
                    p->ff_step0 += f0;
                }
                p->ftiles.push_back(t);
            }
        }
        sl.tile_end = (int)p->ftiles.size();
        p->slabs.push_back(sl);
    }
    if (chunks_out) chunks_out->swap(chunks);
    return PPL_OK;
}

// Size the PPL_SYM_FULL buffers for `room` bytes: the host half (geometry, byte counts, chunk table).  Sets full_planned when they
// fit; ppl_plan then allocates them (full_allocate, ppl_api.cu) and sets full_ok, ppl_plan_dry takes the plan as it is.
int full_plan(ppl_plan_s *p, size_t room) {
    p->full_ok = 0;
    if (!p->use_tma || !p->sa_ok || p->v < 2) return PPL_OK;
    const int v = p->vp, TA = ppl::TA_FULL;
    const size_t lpad_bytes = (p->v & 1) ? align256((size_t)p->x * p->vvp * 8) : 0;
    int tbg = p->dbg.full_tbg >= 16 ? p->dbg.full_tbg / 16 * 16 : 256;  // debug override of the largest tile (rows / 16)
    tbg = std::min(tbg, (v + 15) / 16 * 16);
    const size_t racc_bytes = p->tau_bytes;  // same shapes as tau+-
    std::vector<int2> &chunks = p->chunks_host;
    const int want_slots = p->dbg.full_slots == 1 ? 1 : 2;
    const int tbg0 = tbg;
    size_t &x_bytes = p->fx_bytes, &lq_bytes = p->lq_bytes;
    bool &two_strips = p->two_strips;
    bool fits = false;
    p->lpad_bytes = lpad_bytes;
    p->full_planned = 0;
    // First the slab strip (16 v^3 doubles: step 0 on d-block >= b-block only, 1/8 of nominal).  If it does not fit under
    // the cap, the memory-tight mode: a strip of one (slab; b-group) tile (16 tbg v^2), step 0 per tile on the group's
    // full (b, d) rectangle (1/4 of nominal), everything behind the fold unchanged.
    for (int tight = p->dbg.full_tight == 1 ? 1 : 0; tight <= 1 && !fits; ++tight)
        for (tbg = tbg0;; tbg = std::max(16, tbg / 2 / 16 * 16)) {
            x_bytes = align256((size_t)TA * (tight ? tbg : v) * p->vvp * 8);
            // A second strip pays where slabs are short (medium: 26.19 -> 25.82 ms for 1 GB); at large it buys 0.15 % for
            // 8.2 GB and is not taken.  In the tight mode it is what lets step 0 of tile k+1 overlap the GEMMs of tile k.
            const int want_strips = p->dbg.full_strips ? (p->dbg.full_strips == 1 ? 1 : 2) : ((tight || x_bytes <= ((size_t)2 << 30)) ? 2 : 1);
            const size_t slot_rows = (size_t)TA * tbg + 16;  // + 16: the minus run of a range tile may be a few rows longer than the plus run
            const size_t slot = align256(slot_rows * p->ldp * 8) + align256(slot_rows * p->ldm * 8);
            const size_t part_cap = std::max<size_t>((size_t)64 << 20, slot / 8);
            if (full_geometry(p, tbg, part_cap, &chunks, tight != 0) != PPL_OK) {
                p->dbg.full_rect_tiles = 1;  // (never taken: the range tiling failed its own invariants)
                full_geometry(p, tbg, part_cap, &chunks, tight != 0);
            }
            const size_t chunk_bytes = align256(chunks.size() * sizeof(int2));
            lq_bytes = p->diag_pack ? align256((size_t)p->x * p->ldq * 8) : 0;
            const size_t base = x_bytes + align256(p->fpart_bytes) + racc_bytes + chunk_bytes + lpad_bytes + lq_bytes + 256;
            int ns = 0;
            for (int s = want_slots; s >= 1 && !ns; --s)
                if (base + s * slot <= room) ns = s;
            if (ns) {
                p->tbg = tbg;
                p->fslots = ns;
                p->full_tight = tight;
                p->fws_bytes = base + ns * slot;
                two_strips = want_strips == 2 && ns == want_slots && p->fws_bytes + x_bytes <= room;
                if (two_strips) p->fws_bytes += x_bytes;
                fits = true;
                break;
            }
            if (tbg == 16) break;
        }
    if (!fits) return PPL_OK;  // the plan stays without PPL_SYM_FULL
    p->full_planned = 1;       // slabs, tiles, splits and byte counts are final at this point
    return PPL_OK;
}
// The host half of ppl_plan: everything that follows from (nocc, nvirt, nchol), the byte budget `cap`, the SM count and
// the kernel family alone -- packed geometry, row tiling of step 1, tile edge T, ring depth, buffer sizes.  No CUDA call.
ppl_plan_s *plan_host(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t cap, int num_sms, bool use_tma,
                      const ppl_debug_opts_t *dbg, int *rc_out) {
    *rc_out = PPL_OK;
    ppl_plan_s *p = new (std::nothrow) ppl_plan_s();
    if (!p) {
        *rc_out = PPL_ERR_ALLOC;
        return nullptr;
    }
    if (dbg) p->dbg = *dbg;
    p->o = nocc;
    p->v = nvirt;
    p->x = nchol;
    p->num_sms = num_sms;
    p->vec16 = (nvirt % 2 == 0) ? 1 : 0;
    p->vv = (int64_t)nvirt * nvirt;
    p->vp = nvirt + (nvirt & 1);
    p->vvp = (int64_t)p->vp * p->vp;
    p->cap = workspace_bytes;
    p->Mp = nocc * (nocc + 1) / 2;
    p->Mm = nocc * (nocc - 1) / 2;
    p->KpT = p->vp * (p->vp + 1) / 2;         // packed geometry: nvirt rounded up to even (the pad index carries zeros)
    p->KmT = p->vp * (p->vp - 1) / 2;
    p->Kp = (int)ppl::kplus_extent(p->vp);   // extents of the packed index ranges, holes included (ppl_kernels.cuh)
    p->Km = (int)ppl::kminus_extent(p->vp);
    p->ldp = ((int64_t)p->Kp + 15) / 16 * 16;  // rows of the packed operands are 128-byte aligned: TMA-legal for any nvirt
    p->ldm = ((int64_t)std::max(p->Km, 1) + 15) / 16 * 16;
    p->use_tma = use_tma ? 1 : 0;
    const int ni_env = (p->dbg.ni_max >= 1 && p->dbg.ni_max <= 10) ? p->dbg.ni_max : 10;  // largest row-tile instance used
    const bool tma_full = p->use_tma && p->vec16;
    p->mg_full = tma_full ? m_geom_tma(nocc * nocc, ni_env) : m_geom_plain(nocc * nocc);
    p->mg_p = p->use_tma ? m_geom_tma(p->Mp, ni_env) : m_geom_plain(p->Mp);
    p->mg_m = p->use_tma ? m_geom_tma(std::max(p->Mm, 1), ni_env) : m_geom_plain(std::max(p->Mm, 1));
    p->bm_full = tma_full ? 16 * p->mg_full.ni : ppl::BM;
    p->bm_p = p->use_tma ? 16 * p->mg_p.ni : ppl::BM;
    p->bm_m = p->use_tma ? 16 * p->mg_m.ni : ppl::BM;
    Geometry g{p->vv, nocc * nocc, p->Mp, p->Mm, p->Kp, p->Km, p->ldp, p->ldm, p->mg_full, p->mg_p, p->mg_m};
    p->tau_bytes = align256((size_t)p->Mp * p->ldp * 8) + align256((size_t)std::max(p->Mm, 1) * p->ldm * 8);

    // choose the tile edge T (and ring depth) that minimises the estimated apply time under the cap:
    // first with the packed operands of PPL_SYM_PAIR_SA, and if they do not fit, without them
    const int forced_T = p->dbg.tile_edge > 0 ? std::min(p->dbg.tile_edge, nvirt) : 0;  // debug override
    double best_t = 1e300;
    int best_T = 0, best_ring = 1, best_sa = 0;
    PlanEval best_ev;
    for (int sa = 1; sa >= 0 && best_T == 0; --sa)
        for (int T = nvirt; T >= 1; --T) {
            if (forced_T && T != forced_T) continue;
            // only edges that tile v evenly or nearly so (ragged edge at least T/4), to keep edge tiles efficient; the cost model
            // weighs the rest.  (T/2 until round 2: it ruled out T = 16 at nvirt = 900 -- ragged 4 -- and the plan took T = 22, whose
            // 484-row W tiles pad to 512 in step 1: 571 s instead of 549 s on the Table 3 row N = 1000; medium in the un-packed modes
            // moved from T = 30 to 32: 68.2 -> 65.8 ms)
            const int nblk = (nvirt + T - 1) / T;
            const int r = nvirt - (nblk - 1) * T;
            if (!forced_T && nblk > 1 && 4 * r < T) continue;
            const PlanEval ev = evaluate(g, nocc, nvirt, nchol, T, sa != 0, p->num_sms);
            const size_t fixed = ev.x_bytes + ev.part_bytes + (sa ? p->tau_bytes : 0) + 256;
            int ring = 0;
            for (int rg = std::min(3, MAX_RING); rg >= 1; --rg)
                if (rg * ev.slot_bytes + fixed <= cap) {
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
                best_sa = sa;
            }
        }
    // The one-kernel path (ppl_kernels_small.cuh): nvirt <= 56 (W_ab lives in NB x NB accumulator blocks, NB = ceil(nvirt / 8)
    // <= 7: 98 of a thread's 255 registers), nocc <= 8 (step 1 runs as FMAs out of those registers) and a launch-bound amount of work.
    {
        const int NB = (nvirt + 7) / 8, W8 = 8 * NB, nkt = (nchol + ppl::BK - 1) / ppl::BK;
        for (int pair = 0; pair < 2; ++pair) {
            int items = 0;
            int64_t warps = 0;  // (a, b) columns computed
            for (int a = 0; a < nvirt; ++a) {
                const int nb = pair ? nvirt - a : nvirt;
                items += (nb + SMALL_SW_HOST - 1) / SMALL_SW_HOST;
                warps += nb;
            }
            p->small_items[pair] = items;
            p->fs_step0[pair] = 2.0 * (ppl::BK * (double)nkt) * W8 * W8 * warps;  // DMMA, padded to 8-blocks and 16 k
            p->fs_step1[pair] = 2.0 * nocc * nocc * (double)W8 * W8 * warps;       // FMAs out of the accumulators
        }
        p->small_ok = !p->dbg.no_small_fused && nvirt <= 56 && nocc <= 8 && p->fs_step0[1] + p->fs_step1[1] < GRAPH_AUTO_FLOPS;
    }
    if (best_T == 0) {
        delete p;
        *rc_out = PPL_ERR_WORKSPACE_TOO_SMALL;
        return nullptr;
    }
    p->T = best_T;
    p->nblk = (nvirt + best_T - 1) / best_T;
    p->ring = best_ring;
    p->sa_ok = best_sa;
    p->x_bytes = best_ev.x_bytes;
    p->slot_bytes = best_ev.slot_bytes;
    p->part_bytes = best_ev.part_bytes;
    p->ws_bytes = p->x_bytes + p->ring * p->slot_bytes + p->part_bytes + (p->sa_ok ? p->tau_bytes : 0);
    return p;
}

bool dims_ok(int nocc, int nvirt, int nchol) {
    return nocc >= 1 && nvirt >= 1 && nchol >= 1 && (int64_t)nvirt * nvirt <= INT32_MAX / 2 && (int64_t)nocc * nocc <= INT32_MAX / 2;
}

int full_min_v(const ppl_plan_s *p) { return p->dbg.full_min_v > 0 ? p->dbg.full_min_v : 52; }


bool graph_wanted(const ppl_plan_s *p) {
    if (p->small_ok) return false;  // one launch: nothing to replay
    if (p->graph_mode >= 0) return p->graph_mode == 1;
    const double f = p->sym == PPL_SYM_FULL ? p->ff_step0 + p->ff_step1 : p->f_step0 + p->f_step1;
    return f < GRAPH_AUTO_FLOPS;
}

}  // namespace pplh

using namespace pplh;

int ppl_fail_code(int code) { return pplh::fail(code); }  // for the .cu translation units

extern "C" {

int ppl_last_error(void) { return pplh::fail_peek(); }

const char *ppl_error_string(int code) {
    switch (code) {
        case PPL_OK: return "ok";
        case PPL_ERR_INVALID_ARG: return "invalid argument";
        case PPL_ERR_WORKSPACE_TOO_SMALL: return "workspace_bytes below the minimum plan";
        case PPL_ERR_ALLOC: return "allocation failed";
        case PPL_ERR_CUDA: return "CUDA runtime error";
        case PPL_ERR_UNSUPPORTED_DEVICE: return "no CUDA device of compute capability 10.x (no fallback path exists)";
        case PPL_ERR_PRECONDITION: return "input violates a symmetry the plan relies on";
        case PPL_ERR_SCRATCH_LIMIT: return "request exceeds the built-in scratch of the no-allocation entry point (PPL_NOALLOC_SCRATCH_BYTES)";
        default: return "unknown error";
    }
}

// ppl_plan_dry: the planner alone, for a stated device (free bytes, SM count): no CUDA call, nothing allocated.
int ppl_plan_dry(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t device_free_bytes, int num_sms, int mode,
                 ppl_info_t *out) {
    return ppl_plan_dry_ex(nocc, nvirt, nchol, workspace_bytes, device_free_bytes, num_sms, mode, nullptr, out);
}

int ppl_plan_dry_ex(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t device_free_bytes, int num_sms, int mode,
                    const ppl_debug_opts_t *dbg, ppl_info_t *out) {
    if (!out || !dims_ok(nocc, nvirt, nchol) || num_sms < 1 || mode < -1 || mode > PPL_SYM_FULL) return fail(PPL_ERR_INVALID_ARG);
    const size_t auto_cap = (size_t)(0.9 * (double)device_free_bytes);
    const size_t cap = workspace_bytes ? std::min(workspace_bytes, auto_cap) : auto_cap;
    int rc = PPL_OK;
    ppl_plan_s *p = plan_host(nocc, nvirt, nchol, workspace_bytes, cap, num_sms, !(dbg && dbg->cpasync_kernels), dbg, &rc);
    if (!p) return fail(rc);
    p->dry = 1;
    p->sym = p->sa_ok ? PPL_SYM_PAIR_SA : PPL_SYM_PAIR;
    rc = build_tiles(p);
    if (rc == PPL_OK) {
        full_plan(p, cap > p->ws_bytes ? cap - p->ws_bytes : 0);
        p->full_ok = p->full_planned;
        if (p->full_ok && nvirt >= full_min_v(p)) p->sym = PPL_SYM_FULL;
        if (mode >= 0) rc = ppl_plan_set_symmetry(p, mode);
    }
    if (rc == PPL_OK) rc = ppl_plan_info(p, out);
    delete p;  // a dry plan owns nothing on the device
    return rc == PPL_OK ? PPL_OK : fail(rc);
}

int ppl_plan_set_symmetry(ppl_plan_t *p, int mode) {
    if (!p || (mode != PPL_SYM_NONE && mode != PPL_SYM_PAIR && mode != PPL_SYM_PAIR_SA && mode != PPL_SYM_FULL))
        return fail(PPL_ERR_INVALID_ARG);
    if (mode == PPL_SYM_PAIR_SA && !p->sa_ok) return fail(PPL_ERR_WORKSPACE_TOO_SMALL);
    if (mode == PPL_SYM_FULL) {
        if (!p->full_ok) return fail(PPL_ERR_WORKSPACE_TOO_SMALL);
        p->sym = mode;  // the slab / tile lists were built by ppl_plan
        return PPL_OK;
    }
    const int old = p->sym;
    p->sym = mode;
    const int rc = build_tiles(p);
    if (rc != PPL_OK) {
        p->sym = old;
        build_tiles(p);
        return fail(rc);
    }
    return PPL_OK;
}

int ppl_plan_info(const ppl_plan_t *p, ppl_info_t *out) {
    if (!p || !out) return fail(PPL_ERR_INVALID_ARG);
    memset(out, 0, sizeof(*out));
    const bool sa = p->sym == PPL_SYM_PAIR_SA;
    out->nocc = p->o;
    out->nvirt = p->v;
    out->nchol = p->x;
    out->symmetry = p->sym;
    out->ta = out->tb = p->T;
    out->n_ablocks = out->n_bblocks = p->nblk;
    out->n_tiles = (int)p->tiles.size();
    out->ring = p->ring;
    out->splitk = p->tiles.empty() ? 0 : (sa ? p->tiles[0].sp.splitk : p->tiles[0].full.splitk);
    out->vec16 = p->vec16;
    const bool minus = p->Mm > 0 && p->Km > 0;
    out->launches_per_apply = sa ? 1 + (minus ? 5 : 4) * (int)p->tiles.size() : 3 * (int)p->tiles.size();
    out->step1_tile_m = sa ? p->bm_p : p->bm_full;
    out->workspace_bytes = p->ws_bytes;
    const double v4 = std::pow((double)p->v, 4);
    out->flops_nominal = 2.0 * p->x * v4 + 2.0 * p->o * p->o * v4;
    out->flops_step0 = p->f_step0;
    out->flops_step1 = p->f_step1;
    out->flops_executed = p->f_step0 + p->f_step1;
    out->sa_splitk_plus = p->tiles.empty() ? 0 : p->tiles[0].sp.splitk;
    out->sa_splitk_minus = p->tiles.empty() ? 0 : p->tiles[0].sm.splitk;
    out->sa_tile_m_plus = p->bm_p;
    out->sa_tile_m_minus = p->bm_m;
    out->sa_rows_plus = p->Mp;
    out->sa_rows_minus = p->Mm;
    out->sa_k_plus = p->KpT;
    out->sa_k_minus = p->KmT;
    {   // useful flops of the mode (include/ppl.h): exact pair counts, no padding, no zero rows, no overshoot
        const double v = p->v, P2 = v * (v + 1) / 2, Q2 = v * (v - 1) / 2, M = (double)p->o * p->o;
        const double Mp = p->Mp, Mm = p->Mm;
        switch (p->sym) {
            case PPL_SYM_FULL:
                out->flops_useful_step0 = 2.0 * p->x * P2 * (P2 + 1) / 2;
                out->flops_useful_step1 = 2.0 * (Mp * P2 * P2 + Mm * Q2 * Q2);
                break;
            case PPL_SYM_PAIR_SA:
                out->flops_useful_step0 = 2.0 * p->x * v * v * P2;
                out->flops_useful_step1 = 2.0 * (Mp * P2 + Mm * Q2) * P2;
                break;
            case PPL_SYM_PAIR:
                out->flops_useful_step0 = 2.0 * p->x * v * v * P2;
                out->flops_useful_step1 = 2.0 * M * v * v * P2;
                break;
            default:
                out->flops_useful_step0 = 2.0 * p->x * v4;
                out->flops_useful_step1 = 2.0 * M * v4;
        }
        out->flops_useful = out->flops_useful_step0 + out->flops_useful_step1;
    }
    out->small_fused = p->small_ok;
    out->full_available = p->full_ok;
    out->full_tbg = p->tbg;
    out->full_slabs = (int)p->slabs.size();
    out->full_tight = p->full_ok ? p->full_tight : 0;
    out->full_workspace_bytes = p->fws_bytes;
    out->workspace_bytes = p->ws_bytes + p->fws_bytes;
    if (p->sym == PPL_SYM_FULL) {
        out->ta = ppl::TA_FULL;
        out->tb = p->tbg;
        out->n_ablocks = (int)p->slabs.size();
        out->n_bblocks = p->slabs.empty() ? 0 : p->slabs[0].tile_end - p->slabs[0].tile_begin;
        out->n_tiles = (int)p->ftiles.size();
        out->ring = 1;
        out->splitk = p->ftiles.empty() ? 0 : p->ftiles[0].sp.splitk;
        // pack, unpack, one step 0 per slab -- per tile in the memory-tight mode -- (+ the L pad copy for odd nvirt)
        int launches = 2 + (int)(p->full_tight ? p->ftiles.size() : p->slabs.size()) + ((p->v & 1) ? 1 : 0) +
                       ((p->diag_pack && !p->full_tight) ? 1 : 0);
        for (const FullTile &t : p->ftiles) {
            const int Nm = t.range ? t.nm : ppl::TA_FULL * t.tbp;
            const bool m1 = minus && p->Km - t.k0m > 0 && Nm > 0;
            launches += 1 + (m1 ? 4 : 2) + (p->Kp - t.k1p > 0 ? 1 : 0) + (minus && p->Km - t.k1m > 0 && Nm > 0 ? 1 : 0);
        }
        out->launches_per_apply = launches;
        out->step1_tile_m = p->bm_p;
        out->flops_step0 = p->ff_step0;
        out->flops_step1 = p->ff_step1;
        out->flops_executed = p->ff_step0 + p->ff_step1;
        out->sa_splitk_plus = p->ftiles.empty() ? 0 : p->ftiles[0].sp.splitk;
        out->sa_splitk_minus = p->ftiles.empty() ? 0 : p->ftiles[0].sm.splitk;
    }
    if (p->small_ok) {  // what ppl_apply actually runs: one launch, pair symmetry when the mode allows it
        const int pr = p->sym != PPL_SYM_NONE ? 1 : 0;
        out->n_tiles = p->small_items[pr];
        out->launches_per_apply = 1 + ((p->v & 1) ? 1 : 0);  // + the copy into even-length rows for odd nvirt (also taken for 'iajb' t2 / misaligned buffers)
        out->ring = 1;
        out->splitk = 1;
        out->flops_step0 = p->fs_step0[pr];
        out->flops_step1 = p->fs_step1[pr];
        out->flops_executed = out->flops_step0 + out->flops_step1;
    }
    return PPL_OK;
}

int ppl_plan_set_graph(ppl_plan_t *p, int mode) {
    if (!p || mode < -1 || mode > 1) return fail(PPL_ERR_INVALID_ARG);
    p->graph_mode = mode;
    return PPL_OK;
}

int ppl_plan_set_option(ppl_plan_t *p, int option, int value) {
    if (!p) return fail(PPL_ERR_INVALID_ARG);
    switch (option) {
        case PPL_OPT_VERIFY_INPUTS:
            if (value < 0 || value > 2) return fail(PPL_ERR_INVALID_ARG);
            p->verify = value;
            return PPL_OK;
        default: return fail(PPL_ERR_INVALID_ARG);
    }
}

}  // extern "C"
