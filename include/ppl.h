/*
 * ppl.h -- C ABI of libppl: the CCSD particle-particle ladder contraction with
 * Cholesky-decomposed ERIs on one NVIDIA B200 (sm_100a), FP64.
 *
 *     R[i,j,a,b] += sum_{c,d} (ac|bd) * t2[i,j,c,d],      (ac|bd) = sum_P L[P,a,c] * L[P,b,d]
 *
 * Source of the operation (arxiv/paper_2603_20912, line numbers in /root/reference/PAPER.md):
 *   eq. (4) l.58   pp-ladder term  sum_cd <ab|cd> t_ij^cd, the O(o^2 v^4) bottleneck of CCD/CCSD
 *   eq. (5) l.63   <ab|cd> ~= sum_x L^x_ac L^x_bd  (one L array serves both factors, l.66)
 *   eq. (6) l.68   t~_ij^ab = ... + sum_{x,c,d} L^x_ac L^x_bd t_ij^cd + ...
 *   l.71-73, 118-120   evaluated through the v^4 intermediate in two steps:
 *                      step 0 'xac,xbd->acbd'   (GEMM over the Cholesky index x = P)
 *                      step 1 'acbd,ecfd->efab' (GEMM over (c,d)), result ACCUMULATED (l.177, 331)
 * The v^4 intermediate W = (ac|bd) is never stored whole: it is produced one (a-block x b-block
 * x all c,d) tile at a time into a ring in the plan's workspace and consumed at once.
 *
 * Conventions
 *   - All arrays are dense, row-major FP64 (IEEE binary64) with no strides:
 *         L [nchol][nvirt][nvirt]            Cholesky vectors, L[P][a][c]
 *         t2[nocc][nocc][nvirt][nvirt]       amplitudes,       t2[i][j][c][d]
 *         R [nocc][nocc][nvirt][nvirt]       result,           R[i][j][a][b]   (in/out)
 *   - Semantics: accumulate, coefficient exactly 1 (eq. 6 has no prefactor).  The caller zeroes R
 *     if it wants the bare term.  R must not alias L or t2.
 *   - Ownership: the plan owns its workspace, internal stream and events.  L, t2, R are borrowed.
 *   - Errors: every entry point returns a PPL_* code (ppl_plan returns NULL and records the code
 *     for ppl_last_error()).  No exceptions, no exit(), NO CPU FALLBACK: on anything but a
 *     compute-capability 10.x device the library refuses (PPL_ERR_UNSUPPORTED_DEVICE).
 *   - Threading: one in-flight ppl_apply per plan (the workspace is shared); distinct plans are
 *     independent.  ppl_last_error() is per thread.
 *   - Devices: a plan belongs to the CUDA device that was current when ppl_plan ran (its workspace, streams and
 *     events live there).  Every entry point that takes a plan returns PPL_ERR_INVALID_ARG when the calling
 *     thread's current device is another one; make the plan's device current first (cudaSetDevice).
 */
#ifndef PPL_H
#define PPL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ppl_plan_s ppl_plan_t; /* opaque */

enum {
    PPL_OK = 0,
    PPL_ERR_INVALID_ARG = 1,         /* NULL / non-positive dimension / misaligned pointer */
    PPL_ERR_WORKSPACE_TOO_SMALL = 2, /* workspace_bytes below the minimum plan */
    PPL_ERR_ALLOC = 3,               /* cudaMalloc / host allocation failed */
    PPL_ERR_CUDA = 4,                /* a CUDA runtime call or kernel launch failed */
    PPL_ERR_UNSUPPORTED_DEVICE = 5,  /* no CUDA device, or not compute capability 10.x */
    PPL_ERR_PRECONDITION = 6,        /* ppl_check_inputs: a symmetry the plan relies on is violated */
    PPL_ERR_SCRATCH_LIMIT = 7        /* ppl_contract_pair_noalloc: the request needs more than PPL_NOALLOC_SCRATCH_BYTES */
};

/* Symmetry modes (ppl_plan_set_symmetry). */
enum {
    PPL_SYM_NONE = 0, /* general t2: every (a-block, b-block) tile is computed */
    PPL_SYM_PAIR = 1, /* t2[i,j,c,d] == t2[j,i,d,c] (holds for CC amplitudes): then
                         R_term[i,j,a,b] == R_term[j,i,b,a] for ANY L, so only tiles with
                         a-block <= b-block are computed and the result is also written into
                         the mirrored entries.  Result undefined if t2 is not pair-symmetric
                         (ppl_check_inputs detects that). */
    PPL_SYM_PAIR_SA = 2,/* same precondition as PPL_SYM_PAIR, and the same tiles; in addition step 1
                         runs on symmetric / antisymmetric packed operands
                             W+-[(ab)][(c<=d)] = (ac|bd) +- (ad|bc),  tau+-[(i<=j)][(c<=d)] = (t2[ij,cd] +- t2[ij,dc])/2,
                             R[i,j,a,b] = R+ + R-,  R[j,i,a,b] = R+ - R-,
                         which halves the flops of step 1 again (an identity for ANY L; SURVEY.md 8(f)
                         NEXT-4, pinned on the CPU by tests/test_oracle_pins.py). */
    PPL_SYM_FULL = 3    /* preconditions: t2 pair-symmetric AND L[P,a,c] == L[P,c,a] (real orbitals, PAPER.md:66;
                         both named by north_star).  Then (ac|bd) has the full 8-fold symmetry and
                             S+-[(a<=b)][(c<=d)] = (ac|bd) +- (ad|bc)
                         is a SYMMETRIC matrix in its two pair indices: only its blocks on or above the diagonal
                         are generated (a-blocks of 16; for slab A all of b, c, d >= A), each used twice
                         (R+-[.][(ab)] += tau+-[.][(cd)] S[(ab)][(cd)] and R+-[.][(cd)] += tau+-[.][(ab)] S[(ab)][(cd)]),
                         and step 0 computes only (ac|bd) with d-block >= b-block.  Executed flops: step 0 ~ 1/8,
                         step 1 ~ 1/4 of nominal.  Result undefined if a precondition is violated
                         (ppl_check_inputs detects both).  Even nvirt: L must be 16-byte aligned (TMA reads it in
                         place).  Odd nvirt: the path runs in the geometry of nvirt + 1 -- L is copied per apply into
                         a plan-owned [nchol][nvirt+1][nvirt+1] buffer with a zero pad row / column,
                         the pad index of the packed operands carries exact zeros and never reaches R.  Its
                         buffers (a 16 x nvirt^3 strip and the R+- accumulators) are allocated by ppl_plan when
                         they fit under the workspace cap.  Default when available and nvirt >= 52. */
};

/* Storage orders of the 4-index arrays t2 and R. */
enum {
    PPL_LAYOUT_IJAB = 0, /* [i][j][c][d] / [i][j][a][b]: BASELINE.json's layout, the paper's 'efab' */
    PPL_LAYOUT_IAJB = 1  /* [i][c][j][d] / [i][a][j][b]: the paper's 'icjd' and 'iajb' */
};

/* Options of ppl_apply_ex.  R = beta * R + alpha * term.  beta == 0 overwrites: R is not read and
 * may be uninitialised.  The permutations are folded into the packing / reduction kernels'
 * addressing (the paper pays a transpose for them). */
typedef struct ppl_opts_s {
    int32_t t2_layout; /* PPL_LAYOUT_* of t2 */
    int32_t r_layout;  /* PPL_LAYOUT_* of R  */
    double alpha;      /* 1.0 in ppl_apply */
    double beta;       /* 1.0 in ppl_apply (accumulate) */
} ppl_opts_t;

/* What the planner chose; filled by ppl_plan_info.  Flop counts follow BASELINE.json:
 * F_nom = 2*nchol*nvirt^4 + 2*nocc^2*nvirt^4; F_exec counts the tiles actually executed. */
typedef struct ppl_info_s {
    int32_t nocc, nvirt, nchol;
    int32_t symmetry;          /* PPL_SYM_* */
    int32_t ta, tb;            /* tile edge lengths along a and b (virtual indices per block) */
    int32_t n_ablocks, n_bblocks;
    int32_t n_tiles;           /* tiles executed per apply */
    int32_t ring;              /* W-tile ring depth */
    int32_t splitk;            /* split-K factor of step 1 (the (c,d) contraction) */
    int32_t vec16;             /* 1: 16-byte async copies (nvirt even); 0: 8-byte path */
    int32_t launches_per_apply;/* kernels launched by one ppl_apply */
    int32_t step1_tile_m;      /* CTA tile rows of step 1 (16*NI chosen to tile nocc^2 with least padding) */
    uint64_t workspace_bytes;  /* device bytes owned by the plan */
    double flops_nominal;      /* F_nom */
    double flops_executed;     /* F_exec: the GEMM extents actually launched, step 0 + step 1 -- INCLUDING what the launches spend
                                  on CTA-tile padding, pad chunks, structurally zero rows and slab-granularity overshoot
                                  (the hardware-rate numerator; compare with flops_useful below) */
    double flops_step0;        /* executed flops of step 0 ('xac,xbd->acbd') */
    double flops_step1;        /* executed flops of step 1 ('acbd,ecfd->efab') */
    int32_t sa_splitk_plus, sa_splitk_minus; /* PPL_SYM_PAIR_SA: split-K of the + / - GEMMs (first tile) */
    int32_t sa_tile_m_plus, sa_tile_m_minus; /* PPL_SYM_PAIR_SA: CTA tile rows of the + / - GEMMs */
    int32_t sa_rows_plus, sa_rows_minus;     /* nocc(nocc+1)/2, nocc(nocc-1)/2 */
    int32_t sa_k_plus, sa_k_minus;           /* v'(v'+1)/2, v'(v'-1)/2, v' = nvirt rounded up to even */
    int32_t full_available;                  /* 1: ppl_plan allocated the PPL_SYM_FULL buffers */
    int32_t full_tbg;                        /* PPL_SYM_FULL: b-group width (tile = 16 a's x full_tbg b's) */
    int32_t full_slabs;                      /* PPL_SYM_FULL: number of a-blocks of 16 (one step-0 launch each) */
    int32_t full_tight;                      /* PPL_SYM_FULL buffers are the memory-tight kind: a strip of one (slab; b-group)
                                                tile instead of the slab's 16 nvirt^3, step 0 per tile at 1/4 of nominal */
    uint64_t full_workspace_bytes;           /* part of workspace_bytes that belongs to PPL_SYM_FULL */
    /* Useful flops: what the symmetry the mode exploits leaves to compute, with no tile padding, no zero rows and no
     * slab-granularity overshoot -- the figure flops_executed is to be compared with (bench.py prints both rates).
     *   PPL_SYM_FULL:    step 0  2 nchol U, U = P (P + 1) / 2 unique (ac|bd) of the 8-fold symmetry, P = nvirt (nvirt + 1) / 2;
     *                    step 1  2 (M+ K+^2 + M- K-^2): the whole symmetric S+- matrices applied once
     *                    (M+- = nocc (nocc +- 1) / 2 rows, K+- = nvirt (nvirt +- 1) / 2 packed pairs)
     *   PPL_SYM_PAIR_SA: step 0  2 nchol nvirt^2 P (W rows a <= b only);  step 1  2 (M+ K+ + M- K-) P
     *   PPL_SYM_PAIR:    (2 nchol + 2 nocc^2) nvirt^2 P;   PPL_SYM_NONE: the nominal count. */
    double flops_useful, flops_useful_step0, flops_useful_step1;
    int32_t small_fused;                     /* 1: ppl_apply runs the one-kernel path of launch-bound shapes (nvirt <= 56, nocc <= 8;
                                                csrc/ppl_kernels_small.cuh): step 0, step 1 and the accumulate / mirror in one
                                                launch, W in registers; pair symmetry only (a <= b), whatever the mode allows */
    int32_t reserved_;
} ppl_info_t;

/* Per-stage device times of the most recent profiled apply (ppl_apply_profiled), milliseconds. */
typedef struct ppl_times_s {
    float total_ms;
    float step0_ms;  /* sum over tiles of the W-tile generation kernel */
    float step1_ms;  /* sum over tiles of the (c,d) contraction kernel */
    float reduce_ms; /* sum over tiles of the split-K reduction + accumulate + mirror kernel */
    int32_t n_step0, n_step1, n_reduce; /* launches */
    float fold_ms;   /* PPL_SYM_PAIR_SA: sum over tiles of the W -> W+- fold kernel */
    float pack_ms;   /* PPL_SYM_PAIR_SA: t2 -> tau+- packing (once per apply); other modes: t2 permute if any */
    int32_t n_fold, n_pack;
} ppl_times_t;

/* ppl_plan: choose tile shape, ring depth and split-K for (nocc, nvirt, nchol) and allocate the
 * device workspace once (the analogue of the paper's memory functions, Table 1 l.99-116, and of
 * its "avoid cudaMalloc per batch" remark l.340-342).
 *   nocc, nvirt, nchol >= 1.
 *   workspace_bytes: CAP on device memory the plan may allocate. 0 = automatic (what the
 *     preferred plan needs, at most 90 % of currently free device memory -- cf. the paper's
 *     avail*0.98*0.9, l.107).  If the cap is below the minimum plan (one (a,b) column of W plus
 *     reduction scratch) -> NULL with PPL_ERR_WORKSPACE_TOO_SMALL.
 * Uses the current CUDA device.  Returns NULL on failure (see ppl_last_error). */
ppl_plan_t *ppl_plan(int nocc, int nvirt, int nchol, size_t workspace_bytes);

/* Debug / experiment knobs of the planner and the orchestration, for tests and A/B measurements (they replace the
 * environment variables of round 1; the library reads no environment variable except PPL_TRACE).  All zero = the
 * product's defaults; ppl_plan(...) == ppl_plan_ex(..., NULL).  The struct is copied into the plan. */
typedef struct ppl_debug_opts_s {
    int32_t tile_edge;        /* un-packed modes: force the W-tile edge T (0 = the planner's choice) */
    int32_t ni_max;           /* largest row-tile instance of step 1, 1..10 (0 = 10) */
    int32_t cpasync_kernels;  /* 1 = the cp.async kernels instead of the TMA kernels */
    int32_t full_min_v;       /* smallest nvirt at which PPL_SYM_FULL is the default (0 = 52) */
    int32_t full_tbg;         /* PPL_SYM_FULL: largest W+- tile, in rows / 16 (0 = 256); a multiple of 16 */
    int32_t full_slots;       /* PPL_SYM_FULL: 1 = a single W+- slot (0 = two when they fit) */
    int32_t full_strips;      /* PPL_SYM_FULL: 1 = one strip, 2 = two whenever they fit (0 = the planner's choice) */
    int32_t full_tight;       /* PPL_SYM_FULL: 1 = the memory-tight form even when the slab strip fits */
    int32_t full_rect_tiles;  /* PPL_SYM_FULL: 1 = rectangular (slab; b-group) W+- tiles with their zero rows (the round-1 form;
                                 always used by the memory-tight form) instead of runs of the packed pair index */
    int32_t full_no_diag_pack;/* PPL_SYM_FULL: 1 = diagonal d-blocks of step 0 as 16 plain chunks instead of 9 packed ones */
    int32_t full_serial;      /* PPL_SYM_FULL: 1 = every launch on the caller's stream */
    int32_t debug_sync;       /* 1 = synchronise and report on stderr after every launch */
    int32_t trace;            /* 1 = timeline of one apply on stderr (also: environment variable PPL_TRACE) */
    int32_t host_chunk_mb;    /* ppl_apply_host: staging-buffer size in MiB (0 = 1024) */
    int32_t no_small_fused;   /* 1 = never take the one-kernel path of launch-bound shapes (nvirt <= 56, nocc <= 8): the tiled
                                 path of the plan's symmetry mode runs instead (tests of the tiled kernels at small shapes) */
    int32_t host_panels;      /* ppl_apply_host, un-packed modes: 1 = stream L as row panels even when L fits on the device whole,
                                 2 = never (L whole or PPL_ERR_ALLOC); 0 = panels only when L does not fit beside t2 */
    int32_t full_group_m;     /* PPL_SYM_FULL, step 0: row tiles per raster group (0 = 12) */
    int32_t full_hints;       /* PPL_SYM_FULL, step 0: L2 policy, a bit mask: 1 = evict_last on the row-panel loads, 2 = evict_first
                                 on the column-panel loads, 4 = streaming (evict-first) stores of the strip, 8 = 128-byte instead
                                 of 256-byte L2 promotion of the TMA loads of L; 0 = the default (1 + 4 + 8), -1 = none */
    int32_t reserved[14];     /* must be zero */
} ppl_debug_opts_t;

/* ppl_plan with debug options (NULL = defaults). */
ppl_plan_t *ppl_plan_ex(int nocc, int nvirt, int nchol, size_t workspace_bytes, const ppl_debug_opts_t *dbg);

/* ppl_apply: enqueue  R += ladder(L, t2)  on `stream` (a cudaStream_t passed as void*; NULL =
 * the legacy default stream).  Asynchronous: returns once the work is queued.  All effects are
 * ordered after prior work on `stream` and complete before later work on `stream` (an internal
 * producer stream is forked and joined with events).
 *   L, t2, R: DEVICE pointers, layouts above, 8-byte aligned (16-byte aligned enables the fast
 *   copy path when nvirt is even; torch allocations are 512-byte aligned).  They must stay valid
 *   until the queued work completes.
 * PRECONDITIONS OF THE DEFAULT MODE: a plan for nvirt >= 52 defaults to PPL_SYM_FULL, which requires the real-orbital
 *   symmetry L[P,a,c] == L[P,c,a] AND pair-symmetric amplitudes t2[i,j,c,d] == t2[j,i,d,c]; below that
 *   the default is PPL_SYM_PAIR_SA, which requires the latter.  Both hold for CC amplitudes and real orbitals, neither
 *   for arbitrary arrays (e.g. the unstructured random arrays of the paper's own benchmark): call
 *   ppl_plan_set_symmetry(plan, PPL_SYM_NONE) for those.  By default every apply verifies the preconditions on the
 *   device (PPL_OPT_VERIFY_INPUTS above) and a violation surfaces as PPL_ERR_PRECONDITION. */
int ppl_apply(ppl_plan_t *plan, const double *L, const double *t2, double *R, void *stream);

/* ppl_apply_ex: ppl_apply with options (storage orders of t2 and R, alpha, beta); opts == NULL
 * means the defaults of ppl_apply.  Same stream semantics.  In the un-packed modes
 * (PPL_SYM_NONE / PPL_SYM_PAIR) a t2 given as PPL_LAYOUT_IAJB is first permuted into a plan-owned
 * buffer (allocated on first use, nocc^2 nvirt^2 doubles); in PPL_SYM_PAIR_SA the packing kernel
 * reads either order in place. */
int ppl_apply_ex(ppl_plan_t *plan, const double *L, const double *t2, double *R, const ppl_opts_t *opts,
                 void *stream);

/* ppl_generate_eri: step 0 alone (the paper's 'xac,xbd->acbd'; eq. 5) -- the dense
 * integrals of a slab of a's in the order the paper's dense variant consumes them ('abcd'):
 *     eri[a-a0][b][c][d] = <ab|cd> = (ac|bd) = sum_P L[P,a,c] * L[P,b,d],   a0 <= a < a0+na, all b, c, d
 * eri is a DEVICE buffer of na * nvirt^3 doubles, overwritten; L as in ppl_apply.  No symmetry of L is assumed or
 * used; nocc of the plan is ignored.  ppl_generate_eri followed by ppl_apply_dense on the same slab equals the
 * slab's share of ppl_apply (the dense / Cholesky duality of PAPER.md:75).  Asynchronous on `stream`.
 * PPL_ERR_INVALID_ARG for a slab outside [0, nvirt) or misaligned pointers. */
int ppl_generate_eri(ppl_plan_t *plan, const double *L, int a0, int na, double *eri, void *stream);

/* ppl_apply_dense: step 1 alone on caller-supplied dense integrals (the
 * paper's 'abcd,ecfd->efab'):
 *     R[i,j,a,b] = beta*R[i,j,a,b] + alpha * sum_{c,d} eri[a-a0][b][c][d] * t2[i,j,c,d],   a0 <= a < a0+na, all b
 * eri is a DEVICE slab [na][nvirt][nvirt][nvirt] of <ab|cd> (physicist order, as the paper's
 * 'abcd'), i.e. exactly the [(a,b)][(c,d)] matrix step 1 consumes.  No symmetry is assumed or
 * used.  nchol of the plan is ignored.  Only R entries with a in the slab are touched. */
int ppl_apply_dense(ppl_plan_t *plan, const double *eri, int a0, int na, const double *t2, double *R,
                    const ppl_opts_t *opts, void *stream);

/* ppl_contract_pair: the generic pair contraction of the paper's generic recipe (pseudo-code 211-338;
 * SURVEY.md 8(f) NEXT-3):
 *     C[out] = beta * C[out] + alpha * sum_{summed letters} A[op0] * B[op1]
 * subscripts: "op0,op1->out", one ASCII letter per axis (at most 12 per operand), no letter repeated inside an operand,
 *   every letter in exactly TWO of op0, op1, out (a tensordot: surviving letters of op0, surviving letters of op1,
 *   summed letters; `out` may order the surviving letters in any way).  Examples: the ladder's own steps
 *   "xac,xbd->acbd" and "abcd,ecfd->efab", "xac,icjd->xajd", "ik,kj->ij".
 * dims0 / dims1: extents of the axes of A / B in the order of op0 / op1 (a shared letter must agree).
 * A, B, C: DEVICE pointers, dense row-major FP64 in the order of their subscripts, 8-byte aligned (16-byte aligned
 *   operands with even extents along their unit-stride letter take the 16-byte copy path).  C must not alias A or B.
 *   beta == 0 overwrites: C is not read.
 * workspace: DEVICE memory, 256-byte aligned, at least the bytes ppl_contract_pair_workspace reports (offset tables of
 *   8 (2 M + 2 N + 2 K) bytes plus room for split-K partials; with less than the report -- but at least the tables --
 *   the call lowers its split-K factor instead of failing).  Borrowed until the queued work completes.
 * Where the paper batches along the surviving axes to fit VRAM and calls tensordot (permuted copies + DGEMM) per batch,
 * this is one in-place GEMM over offset tables on the FP64 tensor pipe; the summed axes (the Cholesky index among them)
 * are split only inside the kernel, with a fixed-order reduction: results are bit-reproducible.  No symmetry is assumed.
 * Asynchronous on `stream`: a call is kernel launches only -- the offset tables are computed on the device from the extents
 * and strides of the axes (no host table, no upload), and the per-device facts (SM count, kernel attributes) are looked up on
 * the first call on a device and cached (thread-safe); make that first call outside any stream capture, later calls may be
 * captured into a CUDA graph (tests/test_gpu_contract.py).  Needs no plan.  PPL_ERR_INVALID_ARG for a malformed request,
 * PPL_ERR_WORKSPACE_TOO_SMALL if the workspace cannot hold the tables, PPL_ERR_UNSUPPORTED_DEVICE off cc 10.x. */
int ppl_contract_pair_workspace(const char *subscripts, const int64_t *dims0, const int64_t *dims1, size_t *bytes);
int ppl_contract_pair(const char *subscripts, const int64_t *dims0, const int64_t *dims1, const double *A, const double *B,
                      double *C, double alpha, double beta, void *workspace, size_t workspace_bytes, void *stream);

/* ppl_contract_pair_noalloc: ppl_contract_pair for callers that cannot allocate device memory.
 *
 * Who that is: a program that has already handed the whole GPU to its own memory pool (a CC driver that sizes its
 * tensors to 90 % of VRAM the way the paper does; a framework with a caching allocator that owns what is
 * left), so that a cudaMalloc for a workspace would fail or push someone else out; code on a path where cudaMalloc /
 * cudaFree are unwelcome because they synchronise the whole device and take a driver-wide lock; and plug-ins that are
 * handed device pointers and a stream by their host and have no allocator of their own to ask.  Such callers cannot
 * satisfy ppl_contract_pair's `workspace` argument.  This entry point does not have one.
 *
 * Same operation, same arguments otherwise:  C[out] = beta * C[out] + alpha * sum_{summed letters} A[op0] * B[op1],
 * A, B, C DEVICE pointers (8-byte aligned, dense row-major in the order of their subscripts; C must not alias A or B;
 * beta == 0 overwrites without reading C).  It always runs the in-place gather GEMM of the generic recipe (offset
 * tables, DMMA, fixed-order split-K: bit-reproducible); plain matrix pairs are NOT re-routed to the ladder's TMA
 * kernels as in ppl_contract_pair.
 *
 * Scratch: the offset tables, 16 (M + N + K) bytes (M, N = products of the surviving extents of op0 / op1, K = product
 * of the summed extents), and the split-K partials live in a fixed array of PPL_NOALLOC_SCRATCH_BYTES that is part of
 * the library: every GPU on which the library's code is loaded holds those bytes until the process exits, whether or
 * not this function is ever called again.  Apart from the one-time set-up described below, a call is kernel launches
 * only: no cudaMalloc, cudaFree, cudaMemcpy or allocating library routine; the tables are computed on the device.
 *   Limit: a request whose tables alone exceed PPL_NOALLOC_SCRATCH_BYTES is refused with PPL_ERR_SCRATCH_LIMIT and
 *   nothing is queued (use ppl_contract_pair with a workspace of your own).  Partials take what the tables leave:
 *   the split-K factor is lowered, down to none, until they fit -- exactly what ppl_contract_pair does when given a
 *   workspace of PPL_NOALLOC_SCRATCH_BYTES, and with the same results bit for bit on the gather route.
 *   First call on a device: looks up the array's device address and the SM count and opts the kernels into their
 *   shared-memory size, with the calling thread's current device; cached afterwards (thread-safe).  Make that first
 *   call during start-up, before any stream capture begins in the process.
 *   Sharing: there is ONE array per device and every call uses it.  Nothing in it needs clearing between calls (each
 *   call rewrites all it reads), but calls whose kernels may overlap on the GPU -- issued on different streams without
 *   an ordering between them, or from two threads -- race on it and give undefined results.  Calls on one stream, or
 *   ordered by events, are safe.  The array keeps the last call's tables and partials; do not rely on that.
 * Asynchronous on `stream` (NULL = the legacy default stream).  Errors: PPL_ERR_INVALID_ARG (malformed request, NULL or
 * misaligned pointers), PPL_ERR_SCRATCH_LIMIT, PPL_ERR_UNSUPPORTED_DEVICE (no cc 10.x device current),
 * PPL_ERR_CUDA. */
#define PPL_NOALLOC_SCRATCH_BYTES (32u << 20) /* 32 MiB, resident per GPU for the life of the process */
int ppl_contract_pair_noalloc(const char *subscripts, const int64_t *dims0, const int64_t *dims1, const double *A,
                              const double *B, double *C, double alpha, double beta, void *stream);

/* ppl_apply_host: the same operation on HOST buffers (pageable or pinned), the paper's own setting (operands in
 * host memory).  Synchronises before returning.  Device buffers are
 * allocated on first use and kept by the plan (they are not counted against workspace_bytes).
 *   PPL_SYM_FULL: L is copied whole; t2 and R never sit on the device whole -- t2 is streamed through two staging
 *     buffers (1 GiB each) and packed chunk by chunk into tau+-, the slabs run on the packed operands, and R leaves
 *     slab by slab while they run: behind every slab of 16 a's, R[:, :, slab, :] travels in (a 2-D copy), takes the
 *     term, and travels out, beside the GEMMs of the following slabs.  Device residency is about half of L + t2 + R: shapes of the paper's Table 3 fit on one 180 GB GPU.
 *   PPL_SYM_NONE / PPL_SYM_PAIR (nothing assumed of L; PPL_SYM_NONE: nothing of t2 either -- the paper's own benchmark
 *     arrays), even nvirt: t2 is copied whole and stays resident (every W tile contracts with all of it);
 *     L never needs to be: when it does not fit beside t2 it is streamed as row panels L[:, A, :] (a 2-D copy of nchol
 *     rows of |A| nvirt doubles each; the panel of the tile's a-block is kept for a row of tiles, the panel of its b-block
 *     rides a ring of buffers one tile ahead), and in PPL_SYM_NONE R is never on the device whole either: the slab
 *     R[:, :, A, :] of one row of tiles travels in before the row's first reduction and out behind its last, the copies
 *     of row k +- 1 overlapping the GEMMs of row k on streams of their own (in PPL_SYM_PAIR the mirror writes reach
 *     every slab, so R stays resident).  Device residency: t2 + the W ring + a few panels / slabs.
 *   PPL_SYM_PAIR_SA, or odd nvirt: L, t2 and R are copied whole, ppl_apply runs, R is copied back (PPL_ERR_ALLOC if they do not fit).
 *   At shapes that fill the device, plan with workspace_bytes = free device bytes - |L| - 3 GiB - 2 R slabs of 16 a's (nocc^2 x 16 x nvirt doubles each) (what bench.py's
 *   table3_* configs do): the automatic cap of ppl_plan (90 % of the free bytes) leaves no room for L and the staging
 *   buffers, and the call then returns PPL_ERR_ALLOC.  Under such a cap the plan takes the memory-tight form of
 *   PPL_SYM_FULL (ppl_info_t.full_tight) when the 16 nvirt^3 strip does not fit.
 * h2d/d2h byte counts are returned if non-NULL.  R accumulates (+=) as in ppl_apply. */
int ppl_apply_host(ppl_plan_t *plan, const double *L_host, const double *t2_host, double *R_host,
                   uint64_t *h2d_bytes, uint64_t *d2h_bytes);

/* ppl_apply_profiled: like ppl_apply but serialises the stages on `stream`, brackets every
 * kernel with CUDA events, synchronises, and fills *times.  For measurement only. */
int ppl_apply_profiled(ppl_plan_t *plan, const double *L, const double *t2, double *R, void *stream,
                       ppl_times_t *times);

/* ppl_destroy: free the workspace, streams, events and the stored CUDA graph.  NULL is a no-op returning PPL_OK.
 * Synchronises the device first (applies may still be in flight on the caller's streams). */
int ppl_destroy(ppl_plan_t *plan);

/* ---- small extras ------------------------------------------------------------------------- */

int ppl_last_error(void);                /* code of the last failure on this thread */
const char *ppl_error_string(int code);  /* static string, never NULL */

/* Set PPL_SYM_NONE / PPL_SYM_PAIR / PPL_SYM_PAIR_SA / PPL_SYM_FULL.  Default: PPL_SYM_FULL when its
 * buffers fit and nvirt >= 52, else PPL_SYM_PAIR_SA, else PPL_SYM_PAIR if the workspace cap
 * was too small for the packed operands.  PPL_ERR_WORKSPACE_TOO_SMALL if the plan holds no buffers for
 * the requested mode.  Re-plans the tile list; must not be called while an apply is in flight. */
int ppl_plan_set_symmetry(ppl_plan_t *plan, int mode);

/* Plan options.
 * PPL_OPT_VERIFY_INPUTS: what ppl_apply / ppl_apply_ex do about the preconditions of the plan's symmetry mode
 * (PPL_SYM_FULL: L[P,a,c] == L[P,c,a] and t2 pair-symmetric; PPL_SYM_PAIR / PPL_SYM_PAIR_SA: t2 pair-symmetric):
 *   1 (default)  a check kernel is queued at the head of every apply (it reads L and t2 once, coalesced: < 0.1 % of a
 *                call at `large`); the apply itself is queued regardless.  A violation is reported by the NEXT call on
 *                the plan -- ppl_apply*, ppl_plan_verify_status or ppl_destroy -- as PPL_ERR_PRECONDITION (R of the
 *                offending apply is then undefined).  No host synchronisation in the steady state beyond waiting for
 *                that head-of-apply kernel of the previous call.
 *   2            synchronous: the check runs and is awaited first; on a violation nothing else is queued and the call
 *                returns PPL_ERR_PRECONDITION with R untouched.
 *   0            no check: the caller vouches for the preconditions (result undefined otherwise).
 * The check is skipped while the caller is capturing `stream` into a CUDA graph, and in PPL_SYM_NONE (no precondition).
 * On the one-kernel path of launch-bound shapes (ppl_info_t.small_fused) mode 1 costs no launch of its own -- the first CTAs
 * of the apply's single launch scan t2 -- and L is not verified there: that path does not use the symmetry of L, its result
 * is right for any L (mode 2 and ppl_check_inputs verify both arrays as everywhere else).  There the next call reports a
 * violation if the check has finished by then, and otherwise the call after it does: a call never waits for the check of the
 * apply queued just before it (that would serialise host and device at shapes where an apply takes 20 us);
 * ppl_plan_verify_status and ppl_destroy wait for everything outstanding.
 * ppl_apply_host reports a violation from the same call (it synchronises before returning; R is then undefined).  In its
 * streamed PPL_SYM_FULL form t2 never sits on the device whole: its pair symmetry is verified chunk by chunk instead -- the
 * rows i >= j of every staged chunk, which the packing never reads, are folded as their mirror images and compared bit for
 * bit with what the rows (j,i) packed into tau+- (diagonal rows i == j: t2[i,i,c,d] == t2[i,i,d,c] directly). */
enum { PPL_OPT_VERIFY_INPUTS = 1 };
int ppl_plan_set_option(ppl_plan_t *plan, int option, int value);
/* Waits for the check of the most recent apply (if one is pending) and returns PPL_OK or PPL_ERR_PRECONDITION;
 * *flags (if non-NULL): bit 0 = L not symmetric, bit 1 = t2 not pair-symmetric.  Clears the pending state. */
int ppl_plan_verify_status(ppl_plan_t *plan, int *flags);

/* CUDA graph of one apply.  mode 1: ppl_apply / ppl_apply_ex capture the whole apply (all kernels, the forks and
 * joins of the plan's side streams) once into a CUDA graph and replay it with one cudaGraphLaunch on `stream`
 * for as long as (L, t2, R, opts, symmetry mode) stay the same; any change re-captures.  mode 0: plain launches.
 * mode -1 (default): graph when the plan's executed flops are below 5e9 (launch-bound shapes: tiny, small),
 * plain launches above.  If the caller is itself capturing `stream`, the plain launches are issued (and land in
 * the caller's graph) whatever the mode.  ppl_apply_dense, ppl_apply_host and ppl_apply_profiled never use it.
 * Same results bit for bit: the graph holds the same kernels with the same arguments in the same order. */
int ppl_plan_set_graph(ppl_plan_t *plan, int mode);

int ppl_plan_info(const ppl_plan_t *plan, ppl_info_t *out);

/* ppl_plan_dry: the planner alone.  Runs exactly the host half of ppl_plan -- packed geometry, row tiling of step 1,
 * tile edge, ring depth, split-K, slabs / b-groups / strips of PPL_SYM_FULL, buffer sizes, flop accounting -- for a
 * STATED device (free bytes, SM count; the TMA kernel family is assumed) and fills *out as ppl_plan_info would.  No CUDA
 * call, nothing allocated: usable (and tested) on a machine without a GPU.  mode: a PPL_SYM_* value, or -1 for the
 * default ppl_plan would choose.  Errors as ppl_plan / ppl_plan_set_symmetry (PPL_ERR_WORKSPACE_TOO_SMALL ...). */
int ppl_plan_dry(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t device_free_bytes, int num_sms, int mode,
                 ppl_info_t *out);
int ppl_plan_dry_ex(int nocc, int nvirt, int nchol, size_t workspace_bytes, size_t device_free_bytes, int num_sms, int mode,
                    const ppl_debug_opts_t *dbg, ppl_info_t *out);

/* Debug: verify on the device that L[P,a,c]==L[P,c,a] (required in PPL_SYM_FULL, else only reported)
 * and, in every mode but PPL_SYM_NONE, that t2[i,j,c,d]==t2[j,i,d,c] (required).  Synchronises `stream`.
 * Returns PPL_OK, or PPL_ERR_PRECONDITION if an input violates a symmetry the plan relies on.
 * If flags != NULL: bit 0 = L not symmetric, bit 1 = t2 not pair-symmetric. */
int ppl_check_inputs(ppl_plan_t *plan, const double *L, const double *t2, void *stream, int *flags);

/* Measure the FP64 tensor (DMMA, mma.sync.m8n8k4.f64) issue-rate peak of the current device
 * with a register-only kernel: the roofline denominator used by bench.py.  Writes TFLOP/s
 * (best of `reps` launches of about `ms_target` milliseconds each).  Synchronises. */
int ppl_probe_fp64_peak(double *tflops, int reps, double ms_target);

/* The same measurement for the instruction streams the pipe choice was made between (north_star: "FP64 DMMA or the
 * FP64 FMA pipe, whichever ncu shows faster"; evidence in profiles/r02_fp64_peaks.md).  All are register-only loops of
 * 16 warps per SM on every SM; flops counted: 512 per DMMA m8n8k4, 2 per lane per DFMA. */
enum {
    PPL_PROBE_DMMA8 = 0,  /* 8 independent DMMA accumulator chains per warp (ppl_probe_fp64_peak) */
    PPL_PROBE_DMMA16 = 1, /* 16 chains per warp: shows that the 8-chain figure is not dependency-limited */
    PPL_PROBE_DFMA16 = 2, /* plain DFMA, 16 independent chains per thread */
    PPL_PROBE_MIX8 = 3    /* one DFMA per lane interleaved with every DMMA (8 + 8 chains) */
};
int ppl_probe_fp64_pipe(int kind, double *tflops, int reps, double ms_target);

/* Test hook: C(8x8) = A(8x4, row-major) * B(4x8, row-major) through ONE mma.sync.m8n8k4.f64 using
 * the fragment layout the kernels assume (lane = 4g+q: a=A[g][q], b=B[q][g], c={C[g][2q],
 * C[g][2q+1]}).  All three are DEVICE pointers.  Synchronises the device. */
int ppl_debug_dmma_layout(const double *A_dev, const double *B_dev, double *C_dev);

#ifdef __cplusplus
}
#endif
#endif /* PPL_H */
