// ppl_internal.h -- what the translation units of libppl share beyond the plan (ppl_plan.h): error recording and the plain
// GEMM entry points on the persistent TMA kernels (defined in ppl_api.cu, where those kernels are instantiated).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

int ppl_fail_code(int code);  // records the code for ppl_last_error() and returns it (ppl_plan.cpp)

// C[M][N] (dense) = beta C + alpha A^T B,  A[K][M], B[K][N] dense row-major, M and N even, 16-byte aligned bases (k_step0_tma)
int ppl_gemm_kouter_tma(const double *A, const double *B, int M, int N, int K, double *C, double alpha, double beta, int sms,
                        cudaStream_t s);
// part[z][M][N] = split-K partials of A B^T,  A[M][K], B[N][K] dense row-major, K even, 16-byte aligned bases (k_step1_tma)
int ppl_gemm_kinner_tma(const double *A, const double *B, int M, int N, int K, double *part, size_t part_bytes, int *splitk_out,
                        int sms, cudaStream_t s);
