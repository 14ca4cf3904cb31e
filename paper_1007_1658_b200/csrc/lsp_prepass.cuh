// lsp_prepass.cuh -- steps 1-2 of the hot path: normalisation moments and per-sample records.
//
// Step 1: the series is shifted to zero mean and scaled to unit variance.
//   The paper does this on the host before upload; here it is two fp64 device reductions,
//   mean first, then sum (x - mean)^2 fused into the record pass (two-pass variance).
// Step 2 replaces the listing's fp32 `ft = f*t; ft -= rintf(ft)`: fp32 cannot
//   hold frac(f*t) when f*t reaches 1e5 cycles (reading G3).  Each sample gets, ONCE,
//   its phase at f_min and its phase step per frequency bin as exact 64-bit fixed-point turns,
//   plus the rotation (cos, sin) of that step rounded from an fp64 sincospi.
#pragma once
#include "lsp_common.cuh"

namespace lsp {

// Where the time origin goes (reading G6: P does not depend on it, eq. (2)).  The FP32-pipe form steps from one frequency to the
// next with z_{m+1} = 2 cos d_j z_m - z_{m-1}, d_j = 2 pi df t'_j, and the fp32 rounding of 2 cos d_j is an error 6e-8 / sin d_j in
// the step angle, applied K times: samples whose d_j is near 0 or pi carry it.  With the origin at t_0 that is every sample close
// to the start of the series -- all of them on a grid much finer than 1/T.  With the origin 1/(8 df) BEFORE t_0 the step angles
// start at pi/4, and stay inside [pi/4, 3 pi/4] whenever df T <= 1/4 (an oversampling of 4 or more): sin d_j >= 0.71 for every
// sample.  The phases are exact 64-bit turns of the fp64 products, so the longer lever arm costs nothing (bounded to 1e7 cycles
// at the highest frequency, where the fp64 rounding of t' is still 1e-9 cycles).
__host__ __device__ inline double origin_offset(double f_min, double df, int64_t Nf)
{
    const double f_max = f_min + (double)(Nf - 1) * df;
    double off = (df > 0.0) ? 0.125 / df : 0.0;
    if (off * f_max > 1e7) off = 1e7 / f_max;
    return off;
}

// grid (nb, B), any block size (multiple of 32).  part_sum[b][blk] = sum of x over the block's chunk.
// Weighted generalised periodogram (w != NULL): part_sum = sum w x and part_w = sum w over the chunk.
__global__ void moments_kernel(const float* __restrict__ x, int64_t x_stride, int64_t Nt,
                               int64_t chunk, double* __restrict__ part_sum,
                               u64* __restrict__ peak64, unsigned* __restrict__ counter,
                               const float* __restrict__ w = nullptr, int64_t w_stride = 0, double* __restrict__ part_w = nullptr)
{
    __shared__ double red[32];
    const int b = blockIdx.y;
    const float* xb = x + (int64_t)b * x_stride;
    const float* wb = w ? w + (int64_t)b * w_stride : nullptr;
    const int64_t j0 = (int64_t)blockIdx.x * chunk;
    const int64_t j1 = min(Nt, j0 + chunk);
    double acc = 0.0, accw = 0.0;
    for (int64_t j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        if (wb) { const double wj = (double)__ldg(wb + j); acc += wj * (double)__ldg(xb + j); accw += wj; }
        else acc += (double)__ldg(xb + j);
    }
    acc = block_sum(acc, red);
    if (wb) accw = block_sum(accw, red);
    if (threadIdx.x == 0) {
        part_sum[(int64_t)b * gridDim.x + blockIdx.x] = acc;
        if (wb) part_w[(int64_t)b * gridDim.x + blockIdx.x] = accw;
        if (blockIdx.x == 0) { peak64[b] = 0ull; counter[b] = 0u; }
    }
}

// Record order of the tensor-core forms.  The sums of eq. (8) do not care in which order the samples are added, the tensor core's
// round-toward-zero accumulator does: with time-sorted samples a strong slow component of the series (a trend, a period of the order of the
// span -- inside the frequency grid or not) makes the running accumulator of a drain window swing far from the window's final value, and
// the truncation loss, which goes with the ulp of the RUNNING value, is not what tc_trunc_comp reads off the final one: 1.1e-4 ... 2e-4 of
// max P on the CTA-pair kernel for a 20-sigma sinusoid of 1.7 cycles per span below the grid (Nt = 250,001; FP32 form 1.1e-5).  So the
// records are written in a golden-ratio stride order: record i = (j S) mod Nt holds sample j, S ~ 0.618 Nt coprime to Nt -- every run of
// consecutive records, hence every drain window and every MMA, then holds samples from all over the span (three-distance theorem: gaps of
// ~Nt / run), the slow component enters each window with both signs and the accumulator does a random walk.  Costs one scattered 32-byte
// write per sample in the pre-pass.
__host__ inline int64_t record_order_stride(int64_t Nt)
{
    if (Nt < 64) return 1;
    int64_t s = (int64_t)(0.6180339887498949 * (double)Nt);
    for (;; ++s) {
        int64_t a = s, b = Nt;
        while (b) { const int64_t c = a % b; a = b; b = c; }
        if (a == 1) return s;
    }
}
// Weighted generalised periodogram: records of one series' chunk.  With W = sum w, wn_j = Nt w_j / W (mean weight 1):
//   recA  = {sqrt(wn_j) (x_j - xbar_w), cos d_j, sin d_j, 2 cos d_j}   (measurement pass)
//   recA1 = {sqrt(wn_j),                cos d_j, sin d_j, 2 cos d_j}   (weight pass: sum wn cos, sum wn sin)
//   part_var[b][blk] = sum wn_j (x_j - xbar_w)^2  (so that part_var / (Nt - 1) is the weighted sample variance)
// The accumulate kernel scales its anchors by recA1.x, so both passes form sums of wn_j (...) e^{i theta}.
// grid (nb, B); part_sum / part_w from moments_kernel.
__global__ void records_weighted_kernel(const double* __restrict__ t, int64_t t_stride,
                                        const float* __restrict__ x, int64_t x_stride,
                                        const float* __restrict__ w, int64_t w_stride,
                                        int64_t Nt, int64_t chunk, double f_min, double df,
                                        const double* __restrict__ part_sum, const double* __restrict__ part_w,
                                        float4* __restrict__ recA, float4* __restrict__ recA1, ulonglong2* __restrict__ recB,
                                        double* __restrict__ part_var, double t_off /* origin_offset() */,
                                        int trig /* 0: tensor-core forms, which read only .x of the records: no sincospi */,
                                        int64_t order_stride = 1 /* record_order_stride() */)
{
    __shared__ double red[32];
    const int b = blockIdx.y;
    const int nb = gridDim.x;
    const double* tb = t + (int64_t)b * t_stride;
    const float* xb = x + (int64_t)b * x_stride;
    const float* wb = w + (int64_t)b * w_stride;
    double swx = 0.0, sw = 0.0;                            // fixed-order sums of the block partials
    for (int i = 0; i < nb; ++i) { swx += part_sum[(int64_t)b * nb + i]; sw += part_w[(int64_t)b * nb + i]; }
    const double mean = swx / sw;
    const double wscale = (double)Nt / sw;
    const double t0 = __ldg(tb) - t_off;
    const int64_t j0 = (int64_t)blockIdx.x * chunk;
    const int64_t j1 = min(Nt, j0 + chunk);
    double acc = 0.0;
    for (int64_t j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double d = (double)__ldg(xb + j) - mean;
        const double wn = (double)__ldg(wb + j) * wscale;
        acc += wn * d * d;
        const int64_t o = (int64_t)b * Nt + (order_stride == 1 ? j : (int64_t)(((u64)j * (u64)order_stride) % (u64)Nt));
        const double tp = __ldg(tb + j) - t0;
        double vfrac;
        const u64 u = frac_fixed64(f_min, tp, nullptr);
        const u64 v = frac_fixed64(df, tp, &vfrac);
        double sd = 0.0, cd = 0.0;
        if (trig) sincospi(2.0 * vfrac, &sd, &cd);
        const double sq = sqrt(wn);
        recA[o] = make_float4((float)(sq * d), (float)cd, (float)sd, (float)(2.0 * cd));
        recA1[o] = make_float4((float)sq, (float)cd, (float)sd, (float)(2.0 * cd));
        recB[o] = make_ulonglong2(u, v);
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part_var[(int64_t)b * nb + blockIdx.x] = acc;
}

// grid (nb, B).  Writes recA, recB for the block's chunk and part_var[b][blk] = sum (x - mean)^2.
// SHARED (shared-time batch, t_stride = 0): only X_j is needed per series, the phases only once (series 0).
// FUSED (short series, Nt <= 16,384): step 1's sum is formed here -- by EVERY block of the series, over the whole series, with
// the same strided partials and reduction tree, so all blocks hold the identical mean -- and one launch is saved where
// launches are what a call costs (C1, C2, C4); the blocks then share the O(Nt) fp64 record work.
template <bool SHARED, bool FUSED>
__global__ void records_kernel(const double* __restrict__ t, int64_t t_stride,
                               const float* __restrict__ x, int64_t x_stride,
                               int64_t Nt, int64_t chunk, double f_min, double df,
                               double* __restrict__ part_sum,
                               float4* __restrict__ recA, ulonglong2* __restrict__ recB,
                               double* __restrict__ part_var,
                               u64* __restrict__ peak64, unsigned* __restrict__ counter, double t_off /* origin_offset() */,
                               int trig /* 0: tensor-core forms, which read only .x of the records: no sincospi */,
                               int64_t order_stride = 1 /* record i = (j order_stride) mod Nt holds sample j (record_order_stride()) */)
{
    __shared__ double red[32];
    pdl_trigger();                                         // the accumulate kernel may be scheduled now; it waits (pdl_wait) for this grid to finish
    const int b = blockIdx.y;
    const int nb = gridDim.x;
    const double* tb = t + (int64_t)b * t_stride;
    const float* xb = x + (int64_t)b * x_stride;

    double s = 0.0;                                        // fixed-order sum of the block partials
    if (FUSED) {
        double a0 = 0.0;
        for (int64_t j = threadIdx.x; j < Nt; j += blockDim.x) a0 += (double)__ldg(xb + j);
        s = block_sum(a0, red);
        if (threadIdx.x == 0) {                            // part_sum keeps its meaning for later readers: its entries add up to sum x
            part_sum[(int64_t)b * nb + blockIdx.x] = blockIdx.x == 0 ? s : 0.0;
            if (blockIdx.x == 0) { peak64[b] = 0ull; counter[b] = 0u; }
        }
        __syncthreads();                                   // `red` is reused below
    } else
    for (int i = 0; i < nb; ++i) s += part_sum[(int64_t)b * nb + i];
    const double mean = s / (double)Nt;
    const double t0 = __ldg(tb) - t_off;   // time origin (reading G6)

    const int64_t j0 = (int64_t)blockIdx.x * chunk;
    const int64_t j1 = min(Nt, j0 + chunk);
    double acc = 0.0;
    for (int64_t j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double d = (double)__ldg(xb + j) - mean;
        acc += d * d;
        const int64_t o = (int64_t)b * Nt + (order_stride == 1 ? j : (int64_t)(((u64)j * (u64)order_stride) % (u64)Nt));
        if (SHARED && b != 0) continue;                     // shared-time batch: only the variance is needed per series
        const double tp = __ldg(tb + j) - t0;
        double vfrac;
        const u64 u = frac_fixed64(f_min, tp, nullptr);
        const u64 v = frac_fixed64(df, tp, &vfrac);
        double sd = 0.0, cd = 0.0;
        if (!SHARED && trig) sincospi(2.0 * vfrac, &sd, &cd);   // accurate: its error is applied K times per run
        if (!SHARED) recA[o] = make_float4((float)d, (float)cd, (float)sd, (float)(2.0 * cd));
        recB[o] = make_ulonglong2(u, v);
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part_var[(int64_t)b * nb + blockIdx.x] = acc;
}

// Generalised periodogram: a second record array whose "measurement" is the unit weight 1, so that
// the same accumulate kernels return sum cos and sum sin.  n = B * Nt records.
__global__ void unit_records_kernel(const float4* __restrict__ recA, float4* __restrict__ recA1, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { float4 r = recA[i]; r.x = 1.f; recA1[i] = r; }
}

}  // namespace lsp
