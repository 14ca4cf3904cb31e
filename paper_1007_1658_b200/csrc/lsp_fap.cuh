// lsp_fap.cuh -- false-alarm probability of eq. (3) as an elementwise epilogue:
//     Q = 1 - [1 - (1 - p)^((Nt - 3)/2)]^N,    p = 2 P / (Nt - 1),    N = number of independent frequencies
// (the paper writes N_f; PAPER.md:369 replaces it by N_f,ind <= N_f found by Monte-Carlo, so N is a
// real-valued argument).  Reading G13: the paper prints p = 2 P_n / N_t, the beta variable of the law it cites
// when the series is scaled by the N_t-variance; this library scales by the sample variance
// (reading G1), for which the same variable is 2 P / (N_t - 1) -- so Q(P_max) = 0 exactly.  Evaluated in fp64
// through log1p / expm1 so that tiny single-trial probabilities s = (1 - p)^((Nt-3)/2) keep their relative
// accuracy: Q = -expm1(N log1p(-s)).  P and Q may alias (plain loads and stores, no __restrict__).
#pragma once
#include "lsp_common.cuh"

namespace lsp {

__global__ void __launch_bounds__(256) fap_kernel(const float* P, int64_t n, double Nt, double N_ind, float* Q)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double p = (double)P[i];
    double base = 1.0 - 2.0 * p / (Nt - 1.0);              // in [0, 1]: 0 <= P <= (Nt - 1)/2
    base = fmin(fmax(base, 0.0), 1.0);
    const double s = (base > 0.0) ? exp(0.5 * (Nt - 3.0) * log(base)) : 0.0;     // single-trial probability
    const double q = (s < 1.0) ? -expm1(N_ind * log1p(-s)) : 1.0;
    Q[i] = (float)q;
}

}  // namespace lsp
