// A caller of the C ABI that is not Python: plain CUDA runtime + include/ppl.h + libppl.so, no torch.
// Built and run by tests/test_gpu_c_abi.py.  Checks two closed forms that need no oracle:
//   (1) identity-like L (L[P] = s_P * I, symmetric)  =>  (ac|bd) = (sum_P s_P^2) delta_ac delta_bd
//       =>  R = R0 + (sum_P s_P^2) * t2                      (SURVEY 8(c) pin P3; eq. 6)
//   (2) ppl_generate_eri on the same L: eri[a][b][c][d] = (sum_P s_P^2) delta_ac delta_bd
// Exit code 0 on success; prints one line per check.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "ppl.h"

#define CK(call)                                                                  \
    do {                                                                          \
        cudaError_t e__ = (call);                                                 \
        if (e__ != cudaSuccess) {                                                 \
            fprintf(stderr, "%s: %s\n", #call, cudaGetErrorString(e__));          \
            return 2;                                                             \
        }                                                                         \
    } while (0)

int main(int argc, char **argv) {
    const int o = argc > 1 ? atoi(argv[1]) : 6, v = argc > 2 ? atoi(argv[2]) : 64, x = argc > 3 ? atoi(argv[3]) : 24;
    const size_t nL = (size_t)x * v * v, nT = (size_t)o * o * v * v;
    std::vector<double> L(nL, 0.0), t2(nT), R0(nT), R(nT);
    double s2 = 0.0;
    for (int P = 0; P < x; ++P) {
        const double s = 1.0 + 0.25 * P;  // exactly representable, and so is every s^2 and their sum
        s2 += s * s;
        for (int a = 0; a < v; ++a) L[((size_t)P * v + a) * v + a] = s;
    }
    // pair-symmetric t2 of small integers: t2[i,j,c,d] = t2[j,i,d,c]
    for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j)
            for (int c = 0; c < v; ++c)
                for (int d = 0; d < v; ++d) {
                    const int p = i * v + c, q = j * v + d, lo = p < q ? p : q, hi = p < q ? q : p;
                    t2[(((size_t)i * o + j) * v + c) * v + d] = (double)((lo * 7 + hi * 3) % 11 - 5);
                    R0[(((size_t)i * o + j) * v + c) * v + d] = (double)((p * 5 + q) % 13 - 6);
                }
    double *dL, *dT, *dR, *dE;
    CK(cudaMalloc(&dL, nL * 8));
    CK(cudaMalloc(&dT, nT * 8));
    CK(cudaMalloc(&dR, nT * 8));
    CK(cudaMemcpy(dL, L.data(), nL * 8, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(dT, t2.data(), nT * 8, cudaMemcpyHostToDevice));
    cudaStream_t stream;
    CK(cudaStreamCreate(&stream));

    ppl_plan_t *plan = ppl_plan(o, v, x, 0);
    if (!plan) {
        fprintf(stderr, "ppl_plan failed: %s\n", ppl_error_string(ppl_last_error()));
        return 3;
    }
    int bad = 0;
    const int modes[4] = {PPL_SYM_FULL, PPL_SYM_PAIR_SA, PPL_SYM_PAIR, PPL_SYM_NONE};
    for (int m = 0; m < 4; ++m) {
        if (ppl_plan_set_symmetry(plan, modes[m]) != PPL_OK) {
            printf("mode %d not available for this shape: skipped\n", modes[m]);
            continue;
        }
        CK(cudaMemcpyAsync(dR, R0.data(), nT * 8, cudaMemcpyHostToDevice, stream));
        if (ppl_apply(plan, dL, dT, dR, stream) != PPL_OK) {
            fprintf(stderr, "ppl_apply failed: %s\n", ppl_error_string(ppl_last_error()));
            return 4;
        }
        CK(cudaMemcpyAsync(R.data(), dR, nT * 8, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        size_t wrong = 0;
        for (size_t k = 0; k < nT; ++k) wrong += (R[k] != R0[k] + s2 * t2[k]);  // exact: small integers times a dyadic rational
        printf("ppl_apply mode %d: %zu of %zu entries differ from R0 + %.4f * t2\n", modes[m], wrong, nT, s2);
        bad += wrong != 0;
    }
    {
        const int a0 = v / 3, na = v - a0 < 5 ? v - a0 : 5;
        const size_t nE = (size_t)na * v * v * v;
        std::vector<double> E(nE);
        CK(cudaMalloc(&dE, nE * 8));
        CK(cudaMemsetAsync(dE, 0xff, nE * 8, stream));
        if (ppl_generate_eri(plan, dL, a0, na, dE, stream) != PPL_OK) return 5;
        CK(cudaMemcpyAsync(E.data(), dE, nE * 8, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        size_t wrong = 0;
        for (int al = 0; al < na; ++al)
            for (int b = 0; b < v; ++b)
                for (int c = 0; c < v; ++c)
                    for (int d = 0; d < v; ++d) {
                        const double want = (c == a0 + al && d == b) ? s2 : 0.0;
                        wrong += (E[(((size_t)al * v + b) * v + c) * v + d] != want);
                    }
        printf("ppl_generate_eri: %zu of %zu entries differ from %.4f delta_ac delta_bd\n", wrong, nE, s2);
        bad += wrong != 0;
        CK(cudaFree(dE));
    }
    if (ppl_destroy(plan) != PPL_OK) return 6;
    CK(cudaFree(dL));
    CK(cudaFree(dT));
    CK(cudaFree(dR));
    printf(bad ? "C ABI EXAMPLE FAILED\n" : "C ABI EXAMPLE OK\n");
    return bad ? 1 : 0;
}
