// ppl_launch.h -- internal: what ppl_host.cu (host-resident operands) needs from ppl_api.cu, where the kernels are
// instantiated: single launches of the hot-path kernels, the slab loop of PPL_SYM_FULL, the precondition check.
#pragma once
#include "ppl_plan.h"

namespace pplapi {

// 2-D FP64 tensor map {inner (contiguous), outer}, row stride row_bytes, box {box_inner, box_outer}, SWIZZLE_128B, zero fill
int map_2d(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t row_bytes, uint32_t box_inner,
           uint32_t box_outer);

// step 0 of one W tile with the row and the column operand given as two tensor maps {inner = columns, outer = nchol} and
// the first column of the tile's a-block / b-block inside each (the whole L: a0 * nvirt; a row panel of its own: 0)
int step0_tile(const ppl_plan_s *p, const pplh::Tile &t, const CUtensorMap *mapA, int a0v, const CUtensorMap *mapB, int b0v, double *W,
               cudaStream_t s);
// step 1 of one W tile of the un-packed modes out of ring slot `slot` into the plan's split-K partials; mapT: t2 as
// {inner = nvirt^2, outer = nocc^2}, box {BK, step1_tile_m}
int step1_tile(const ppl_plan_s *p, const CUtensorMap *mapT, const double *t2, int slot, const pplh::Tile &t, cudaStream_t s);
// fixed-order sum of the partials into R[i,j,a,b] (+ the mirror if the tile has one); R with element strides (si, sj, sa, sb)
// and r_bias = 0: the caller's array from element (0,0,0,0); a slab buffer that holds only the tile's a-block: its own base
// and r_bias = a0 * sa, the elements the whole array would have in front of it (the kernel subtracts them from the offset)
int reduce_tile(const ppl_plan_s *p, const pplh::Tile &t, double *R, int64_t si, int64_t sj, int64_t sa, int64_t sb, double alpha,
                double beta, cudaStream_t s, int64_t r_bias = 0);
uint32_t step1_box_rows(const ppl_plan_s *p);  // TMA box rows of the t2 map of step1_tile

// PPL_SYM_FULL pieces (ppl_apply_host packs and unpacks chunk by chunk)
// chunk: rows [row0, row1) of t2, row row0 first (the staging buffer itself)
int pack_rows(const ppl_plan_s *p, const double *chunk, double diag, cudaStream_t s, int row0, int row1);
// verification of a staged chunk: its rows i >= j against what the rows i <= j packed (bit 1 of the per-apply flags)
int check_rows(const ppl_plan_s *p, const double *chunk, double diag, cudaStream_t s, int row0, int row1);
int unpack_range(const ppl_plan_s *p, double *R, int64_t idx0, int64_t idx1, cudaStream_t s);
// all slabs on the packed operands.  hook (may be null): called behind the launches of every slab with the two streams whose
// work so far completes the R+-acc columns of that slab's a's [a0, a0 + na)
struct SlabHook {
    int (*fn)(void *ctx, int a0, int na, cudaStream_t s_plus, cudaStream_t s_minus);
    void *ctx;
};
int full_compute(ppl_plan_s *p, const double *L, cudaStream_t s, cudaEvent_t tau_ready, const SlabHook *hook);
// R+-acc -> the slab R[:, :, a0 .. a0 + na, :] held dense in `slab` ([o*o][na][nvirt]); R += term
int unpack_slab(const ppl_plan_s *p, double *slab, int a0, int na, cudaStream_t s);

int verify_begin(ppl_plan_s *p, const double *L, const double *t2, int t2_layout, cudaStream_t stream);
int verify_harvest(ppl_plan_s *p, int *flags_out);

}  // namespace pplapi
