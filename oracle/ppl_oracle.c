/*
 * ppl_oracle.c -- CPU oracle for the CCSD particle-particle ladder with Cholesky-decomposed ERIs.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code with the CUDA path
 * (paper_2603_20912_b200/) and neither includes nor is included by it.  Plain C, FP64, loops in
 * the paper's order; no blocking, fusion or reordering beyond what the definition states.
 *
 * What it computes (the method reaches this definition exactly, up to FP64 summation order):
 *
 *     R[i,j,a,b] += sum_{c,d} ( sum_P L[P,a,c] * L[P,b,d] ) * t2[i,j,c,d]
 *
 *   - eq. (4)  PAPER.md:58   the pp-ladder term  sum_cd <ab|cd> t_ij^cd
 *   - eq. (5)  PAPER.md:63   <ab|cd> ~= sum_x L^x_ac L^x_bd   (a pairs with c, b pairs with d;
 *                            the printed summation index "r" is a garble for x -- reading A1/A2)
 *   - eq. (6)  PAPER.md:68   t~_ij^ab = ... + sum_{x c d} L^x_ac L^x_bd t_ij^cd + ...
 *   - einsum   PAPER.md:75   'xac,xbd,icjd->iajb'  (here stored as L[x,a,c], t2[i,j,c,d],
 *                            R[i,j,a,b] -- BASELINE.json's layout, reading A3)
 *   - route    PAPER.md:71-73, 118-120: the v^4-intermediate route, step 0 'xac,xbd->acbd'
 *                            then step 1 'acbd,ecfd->efab', cost O(x v^4) + O(o^2 v^4)
 *   - "+="     PAPER.md:177, 331 ("add to view of final result array"); coefficient 1 (A4, A5)
 *
 * Layouts: dense row-major, L[nchol][nvirt][nvirt], t2[nocc][nocc][nvirt][nvirt], R like t2.
 * The oracle does NOT assume L[P,a,c] = L[P,c,a] nor t2 pair symmetry: it indexes exactly as
 * written, so it stays valid for non-symmetric test inputs (reading A7).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute force two ways on tiny sizes, a hand-worked
 * 2x2 example (tests/golden/), nchol=1 triple product, identity-L and rank-1-L closed forms, unit
 * impulse (index pairing), linearity / zero / accumulate, output pair symmetry with a negative
 * control, exact-integer inputs against int64 arithmetic, numpy einsum, projection identity.
 * ppl_oracle_eri_slab (step 0 alone) is pinned by a hand-worked example, numpy einsum, the nchol = 1 outer
 * product, the ERI symmetries and by reproducing ppl_oracle_full when contracted with t2.
 * ppl_oracle_contract_pair (the generic two-operand contraction 'op0,op1->out' of PAPER.md:195-209) is the einsum
 * definition written out -- one loop nest over every index letter -- pinned by a hand-worked 2x2x2 example
 * (tests/golden/contract_pair_hand.txt), numpy einsum on the paper's strings and others, matmul / outer-product /
 * trace-free special cases and exact integers.
 * Every entry point below is pinned; none is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int ppl_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* One (a,b) column of the two-step route:
 *   step 0:  Wab[c][d] = sum_P L[P][a][c] * L[P][b][d]          (P ascending)
 *   step 1:  out[ij]  += sum_{c,d} Wab[c][d] * t2[ij][c][d]      ((c,d) ascending)
 * Wab is a caller-provided scratch of v*v doubles; out has stride out_stride between (i,j). */
static void ladder_column(int o, int v, int x, const double *L, const double *t2, int a, int b,
                          double *Wab, double *out, int64_t out_stride) {
    const int64_t vv = (int64_t)v * v;
    memset(Wab, 0, sizeof(double) * (size_t)vv);
    for (int P = 0; P < x; ++P) {
        const double *La = L + (int64_t)P * vv + (int64_t)a * v; /* L[P][a][:] */
        const double *Lb = L + (int64_t)P * vv + (int64_t)b * v; /* L[P][b][:] */
        for (int c = 0; c < v; ++c) {
            const double lac = La[c];
            double *Wc = Wab + (int64_t)c * v;
            for (int d = 0; d < v; ++d) Wc[d] += lac * Lb[d];
        }
    }
    const int64_t oo = (int64_t)o * o;
    for (int64_t ij = 0; ij < oo; ++ij) {
        const double *t = t2 + ij * vv;
        double s = 0.0;
        /* a fixed set of interleaved partial sums (the compiler's SIMD lanes): still one fixed
         * summation order; any order is a valid evaluation of the definition (reading A13) */
#pragma omp simd reduction(+ : s)
        for (int64_t cd = 0; cd < vv; ++cd) s += Wab[cd] * t[cd];
        out[ij * out_stride] += s;
    }
}

/* R[i,j,a,b] += ladder term, every (a,b) column.  Columns write disjoint entries of R, so the
 * OpenMP loop over (a,b) has no races. */
int ppl_oracle_full(int nocc, int nvirt, int nchol, const double *L, const double *t2, double *R) {
    if (nocc < 1 || nvirt < 1 || nchol < 1 || !L || !t2 || !R) return 1;
    const int64_t vv = (int64_t)nvirt * nvirt;
    int fail = 0;
#pragma omp parallel
    {
        double *Wab = (double *)malloc(sizeof(double) * (size_t)vv);
        if (!Wab) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t ab = 0; ab < vv; ++ab) {
                const int a = (int)(ab / nvirt), b = (int)(ab % nvirt);
                ladder_column(nocc, nvirt, nchol, L, t2, a, b, Wab, R + ab, vv);
            }
        }
        free(Wab);
    }
    return fail ? 3 : 0;
}

/* Rcols[p][ij] = ladder term at (a,b) = pairs[p] (bare term: Rcols is overwritten, not
 * accumulated).  Used where the full oracle is unaffordable (large / XL configs). */
int ppl_oracle_columns(int nocc, int nvirt, int nchol, const double *L, const double *t2,
                       int64_t npairs, const int32_t *pairs, double *Rcols) {
    if (nocc < 1 || nvirt < 1 || nchol < 1 || !L || !t2 || npairs < 0) return 1;
    const int64_t vv = (int64_t)nvirt * nvirt, oo = (int64_t)nocc * nocc;
    for (int64_t p = 0; p < npairs; ++p)
        if (pairs[2 * p] < 0 || pairs[2 * p] >= nvirt || pairs[2 * p + 1] < 0 || pairs[2 * p + 1] >= nvirt)
            return 1;
    int fail = 0;
#pragma omp parallel
    {
        double *Wab = (double *)malloc(sizeof(double) * (size_t)vv);
        if (!Wab) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t p = 0; p < npairs; ++p) {
                double *out = Rcols + p * oo;
                memset(out, 0, sizeof(double) * (size_t)oo);
                ladder_column(nocc, nvirt, nchol, L, t2, pairs[2 * p], pairs[2 * p + 1], Wab, out, 1);
            }
        }
        free(Wab);
    }
    return fail ? 3 : 0;
}

/* Brute force (i): materialise the whole W[a][c][b][d] = (ac|bd) (eq. 5) and contract it
 * explicitly with t2 (eq. 4), six nested loops.  Tiny sizes only: v^4 doubles of memory. */
int ppl_oracle_bruteforce_w(int nocc, int nvirt, int nchol, const double *L, const double *t2, double *R) {
    const int64_t o = nocc, v = nvirt, x = nchol;
    double *W = (double *)calloc((size_t)(v * v * v * v), sizeof(double));
    if (!W) return 3;
    for (int64_t a = 0; a < v; ++a)
        for (int64_t c = 0; c < v; ++c)
            for (int64_t b = 0; b < v; ++b)
                for (int64_t d = 0; d < v; ++d) {
                    double s = 0.0;
                    for (int64_t P = 0; P < x; ++P) s += L[(P * v + a) * v + c] * L[(P * v + b) * v + d];
                    W[((a * v + c) * v + b) * v + d] = s;
                }
    for (int64_t i = 0; i < o; ++i)
        for (int64_t j = 0; j < o; ++j)
            for (int64_t a = 0; a < v; ++a)
                for (int64_t b = 0; b < v; ++b) {
                    double s = 0.0;
                    for (int64_t c = 0; c < v; ++c)
                        for (int64_t d = 0; d < v; ++d)
                            s += W[((a * v + c) * v + b) * v + d] * t2[((i * o + j) * v + c) * v + d];
                    R[((i * o + j) * v + a) * v + b] += s;
                }
    free(W);
    return 0;
}

/* Brute force (ii): the direct seven-index sum of eq. (6), no intermediate at all, accumulated in
 * long double (x87 80-bit on x86-64): an independent, more accurate value that also bounds the
 * oracle's own rounding error.  Cost O(x o^2 v^4): tiny sizes only. */
int ppl_oracle_bruteforce_direct(int nocc, int nvirt, int nchol, const double *L, const double *t2, double *R) {
    const int64_t o = nocc, v = nvirt, x = nchol;
#pragma omp parallel for collapse(2) schedule(static)
    for (int64_t i = 0; i < o; ++i)
        for (int64_t j = 0; j < o; ++j)
            for (int64_t a = 0; a < v; ++a)
                for (int64_t b = 0; b < v; ++b) {
                    long double s = 0.0L;
                    for (int64_t P = 0; P < x; ++P)
                        for (int64_t c = 0; c < v; ++c)
                            for (int64_t d = 0; d < v; ++d)
                                s += (long double)L[(P * v + a) * v + c] * (long double)L[(P * v + b) * v + d] *
                                     (long double)t2[((i * o + j) * v + c) * v + d];
                    R[((i * o + j) * v + a) * v + b] += (double)s;
                }
    return 0;
}

/* Projection (Freivalds-style) of the definition, for full-coverage checks at sizes where the
 * full oracle is unaffordable:
 *     sum_{a,b} u[a] w[b] R[i,j,a,b] = sum_{c,d} M[c,d] t2[i,j,c,d],
 *     M[c,d] = sum_P (sum_a u[a] L[P,a,c]) (sum_b w[b] L[P,b,d])
 * which follows from eq. (6) by linearity.  out[ij] is overwritten.  Also returns
 * absout[ij] = sum_cd |M[c,d]| |t2[ij,c,d]| if absout != NULL (a scale for error bounds).
 * long double throughout; cost O(x v^2 + o^2 v^2). */
int ppl_oracle_project(int nocc, int nvirt, int nchol, const double *L, const double *t2, const double *u,
                       const double *w, double *out, double *absout) {
    const int64_t o = nocc, v = nvirt, x = nchol, vv = v * v, oo = o * o;
    long double *M = (long double *)calloc((size_t)vv, sizeof(long double));
    if (!M) return 3;
#pragma omp parallel
    {
        long double *Ml = (long double *)calloc((size_t)vv, sizeof(long double));
        long double *uL = (long double *)malloc(sizeof(long double) * (size_t)v);
        long double *wL = (long double *)malloc(sizeof(long double) * (size_t)v);
#pragma omp for schedule(static)
        for (int64_t P = 0; P < x; ++P) {
            for (int64_t c = 0; c < v; ++c) {
                long double su = 0.0L, sw = 0.0L;
                for (int64_t a = 0; a < v; ++a) {
                    su += (long double)u[a] * (long double)L[(P * v + a) * v + c];
                    sw += (long double)w[a] * (long double)L[(P * v + a) * v + c];
                }
                uL[c] = su;
                wL[c] = sw;
            }
            for (int64_t c = 0; c < v; ++c)
                for (int64_t d = 0; d < v; ++d) Ml[c * v + d] += uL[c] * wL[d];
        }
#pragma omp critical
        for (int64_t k = 0; k < vv; ++k) M[k] += Ml[k];
        free(Ml);
        free(uL);
        free(wL);
    }
#pragma omp parallel for schedule(static)
    for (int64_t ij = 0; ij < oo; ++ij) {
        long double s = 0.0L, sa = 0.0L;
        for (int64_t k = 0; k < vv; ++k) {
            long double p = M[k] * (long double)t2[ij * vv + k];
            s += p;
            sa += p < 0 ? -p : p;
        }
        out[ij] = (double)s;
        if (absout) absout[ij] = (double)sa;
    }
    free(M);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Paper-layout / scaled variant.  The paper stores the amplitudes as
 * 'icjd' and the result as 'iajb' (einsum 'xac,xbd,icjd->iajb'; also written
 * '->efab') and pays a transpose to get there.
 * This entry point evaluates the same definition with either storage order on either side:
 *
 *     R = beta * R + alpha * sum_{c,d} ( sum_P L[P,a,c] L[P,b,d] ) t[i,j,c,d]
 *
 *   layout 0 ("ijab"): element (i,j,p,q) at ((i*o + j)*v + p)*v + q     -- BASELINE.json / 'efab'
 *   layout 1 ("iajb"): element (i,j,p,q) at ((i*v + p)*o + j)*v + q     -- the paper's 'icjd' / 'iajb'
 * beta == 0 means overwrite: R is not read (it may hold NaN).  Same two steps per (a,b) column as
 * ladder_column above, written out again with the index maps so it can be checked by eye.
 * ------------------------------------------------------------------------------------------------ */
static int64_t idx4(int layout, int64_t o, int64_t v, int64_t i, int64_t j, int64_t p, int64_t q) {
    return layout == 0 ? ((i * o + j) * v + p) * v + q : ((i * v + p) * o + j) * v + q;
}

int ppl_oracle_full_ex(int nocc, int nvirt, int nchol, const double *L, const double *t2, double *R,
                       int t2_layout, int r_layout, double alpha, double beta) {
    if (nocc < 1 || nvirt < 1 || nchol < 1 || !L || !t2 || !R) return 1;
    if ((t2_layout != 0 && t2_layout != 1) || (r_layout != 0 && r_layout != 1)) return 1;
    const int64_t o = nocc, v = nvirt, x = nchol, vv = v * v;
    int fail = 0;
#pragma omp parallel
    {
        double *Wab = (double *)malloc(sizeof(double) * (size_t)vv);
        if (!Wab) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t ab = 0; ab < vv; ++ab) {
                const int64_t a = ab / v, b = ab % v;
                /* step 0: Wab[c][d] = sum_P L[P][a][c] L[P][b][d] */
                memset(Wab, 0, sizeof(double) * (size_t)vv);
                for (int64_t P = 0; P < x; ++P)
                    for (int64_t c = 0; c < v; ++c)
                        for (int64_t d = 0; d < v; ++d)
                            Wab[c * v + d] += L[(P * v + a) * v + c] * L[(P * v + b) * v + d];
                /* step 1: one dot product over (c,d) per (i,j) */
                for (int64_t i = 0; i < o; ++i)
                    for (int64_t j = 0; j < o; ++j) {
                        double s = 0.0;
                        for (int64_t c = 0; c < v; ++c)
                            for (int64_t d = 0; d < v; ++d) s += Wab[c * v + d] * t2[idx4(t2_layout, o, v, i, j, c, d)];
                        double *r = R + idx4(r_layout, o, v, i, j, a, b);
                        *r = (beta == 0.0) ? alpha * s : beta * (*r) + alpha * s;
                    }
            }
        }
        free(Wab);
    }
    return fail ? 3 : 0;
}

/* ------------------------------------------------------------------------------------------------
 * Step 0 alone (PAPER.md:118-120 'xac,xbd->acbd'; eq. 5): a slab of the dense integrals
 * in the order the paper's dense variant consumes them ('abcd,ecfd->efab'):
 *
 *     eri[al][b][c][d] = <ab|cd> = (ac|bd) = sum_P L[P][a0+al][c] * L[P][b][d],   0 <= al < na
 *
 * P ascending, plain double accumulation.  No symmetry of L is assumed.  eri is overwritten.
 * Pinned by tests/test_oracle_pins.py (numpy einsum, nchol = 1 outer product bit for bit, the index
 * pairing negative control, and: contracting it with t2 reproduces ppl_oracle_full). */
int ppl_oracle_eri_slab(int nvirt, int nchol, const double *L, int a0, int na, double *eri) {
    if (nvirt < 1 || nchol < 1 || !L || !eri || a0 < 0 || na < 1 || a0 + na > nvirt) return 1;
    const int64_t v = nvirt, x = nchol, vv = v * v;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ab = 0; ab < (int64_t)na * v; ++ab) {
        const int64_t a = a0 + ab / v, b = ab % v;
        double *Wab = eri + ab * vv;
        memset(Wab, 0, sizeof(double) * (size_t)vv);
        for (int64_t P = 0; P < x; ++P)
            for (int64_t c = 0; c < v; ++c)
                for (int64_t d = 0; d < v; ++d)
                    Wab[c * v + d] += L[(P * v + a) * v + c] * L[(P * v + b) * v + d];
    }
    return 0;
}


/* ---------------------------------------------------------------------------------------------
 * Generic pair contraction  'op0,op1->out'  ("any tensor contraction ... translated into a sequence
 * of two-array contractions ... op0,op1->out"; the ladder's own two steps are 'xac,xbd->acbd' and 'abcd,ecfd->efab',
 * PAPER.md:118-120).  The einsum definition, nothing else:
 *
 *     C[out indices] = beta * C[out indices] + alpha * sum_{indices not in out} A[op0 indices] * B[op1 indices]
 *
 * subs: "op0,op1->out", one ASCII letter per axis, no repeated letter inside one operand, every out letter must occur
 * in op0 or op1.  dims0 / dims1: extents of the axes of A / B in the order of op0 / op1 (a letter shared by both must
 * have the same extent).  All arrays dense row-major in the order of their subscripts.  beta == 0 overwrites (C is
 * not read).  One loop nest over the out letters (odometer, row-major), inside it one over the summed letters
 * (odometer in order of first appearance), plain double accumulation.  Returns 0, or 1 on a malformed request.
 * --------------------------------------------------------------------------------------------- */
int ppl_oracle_contract_pair(const char *subs, const int64_t *dims0, const int64_t *dims1, const double *A, const double *B,
                             double *C, double alpha, double beta) {
    char op[3][16];
    int n[3] = {0, 0, 0};
    int which = 0;
    for (const char *q = subs; *q; ++q) {
        if (*q == ',') {
            if (which != 0) return 1;
            which = 1;
        } else if (*q == '-' && q[1] == '>') {
            if (which != 1) return 1;
            which = 2;
            ++q;
        } else if ((*q >= 'a' && *q <= 'z') || (*q >= 'A' && *q <= 'Z')) {
            if (n[which] >= 15) return 1;
            for (int k = 0; k < n[which]; ++k)
                if (op[which][k] == *q) return 1; /* repeated letter inside one operand */
            op[which][n[which]++] = *q;
        } else if (*q != ' ') {
            return 1;
        }
    }
    if (which != 2) return 1;
    int64_t ext[128];
    for (int k = 0; k < 128; ++k) ext[k] = -1;
    for (int k = 0; k < n[0]; ++k) ext[(int)op[0][k]] = dims0[k];
    for (int k = 0; k < n[1]; ++k) {
        if (ext[(int)op[1][k]] >= 0 && ext[(int)op[1][k]] != dims1[k]) return 1;
        ext[(int)op[1][k]] = dims1[k];
    }
    for (int k = 0; k < n[2]; ++k)
        if (ext[(int)op[2][k]] < 0) return 1;
    /* summed letters, in order of first appearance */
    char sum[32];
    int ns = 0;
    for (int w = 0; w < 2; ++w)
        for (int k = 0; k < n[w]; ++k) {
            int seen = 0;
            for (int j = 0; j < n[2]; ++j) seen |= op[2][j] == op[w][k];
            for (int j = 0; j < ns; ++j) seen |= sum[j] == op[w][k];
            if (!seen) sum[ns++] = op[w][k];
        }
    int64_t val[128]; /* current value of every letter */
    for (int k = 0; k < 128; ++k) val[k] = 0;
    int64_t nout = 1, nsum = 1;
    for (int k = 0; k < n[2]; ++k) nout *= ext[(int)op[2][k]];
    for (int k = 0; k < ns; ++k) nsum *= ext[(int)sum[k]];
    for (int64_t io = 0; io < nout; ++io) {
        int64_t r = io; /* row-major odometer of the out letters */
        for (int k = n[2] - 1; k >= 0; --k) {
            val[(int)op[2][k]] = r % ext[(int)op[2][k]];
            r /= ext[(int)op[2][k]];
        }
        double acc = 0.0;
        for (int64_t is = 0; is < nsum; ++is) {
            int64_t q = is;
            for (int k = ns - 1; k >= 0; --k) {
                val[(int)sum[k]] = q % ext[(int)sum[k]];
                q /= ext[(int)sum[k]];
            }
            int64_t ia = 0, ib = 0;
            for (int k = 0; k < n[0]; ++k) ia = ia * dims0[k] + val[(int)op[0][k]];
            for (int k = 0; k < n[1]; ++k) ib = ib * dims1[k] + val[(int)op[1][k]];
            acc += A[ia] * B[ib];
        }
        C[io] = (beta == 0.0) ? alpha * acc : beta * C[io] + alpha * acc;
    }
    return 0;
}
