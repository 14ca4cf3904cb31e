// lsp_refine.cuh -- step 6 for the ill-conditioned frequencies: the six sums again, in fp64, from the raw series.
//
// Eq. (5) divides by (Nt +- R)/2.  Where R -> Nt (f T << 1: every cos^2 is ~1; and the aliases of regular
// sampling) the second term is (S - D)/(Nt - R), a small difference over a small difference: the rounding of the fp32 sums
// of steps 4-5 (relative 1e-7 ... 1e-6 of Nt) is amplified by Nt/(Nt - R).  The generalised periodogram has the same
// structure in its determinant D -> 0.  Such frequencies are few (none on a grid that starts at 1/T unless the sampling is
// regular), so they are simply done again the slow way: one block per frequency, all Nt samples, phases from t (f_min + k df)
// in fp64, fp64 sincospi, fp64 sums in a fixed order -- the arithmetic of the paper's CPU code on the few
// bins that need it.  With fp64 sums the 0/0 decision of reading G7 is taken at the oracle's threshold.
//
// Two users: finish_kernel (lsp_finish.cuh) refines the flagged frequencies of its block in place; the fused epilogues
// (lsp_accum_umma_duo.cuh, lsp_shared_gemm.cuh), which have no block to spare, append (series, frequency) to a bounded
// list that refine_kernel works off afterwards.
#pragma once
#include "lsp_common.cuh"

namespace lsp {

// Which frequencies: those where the rounding of the sums is amplified by more than `amp`, the amplification being
// Nt / (Nt - R) for eq. (5) and (1/4) / D for the generalised form's determinant D <= 1/4 (D ~ (1 - (R/Nt)^2) / 4).
// FP32-pipe form: its sums are good to 1e-7 ... 6e-6 of Nt (the three-term recurrence over K = 32 frequencies at tiny Nt is the
// upper end), so amp = 5 (R > 0.8 Nt) keeps every bin within ~3e-5.
// Tensor-core forms: two error sources grow with R.  (i) sum cos 2 theta, sin 2 theta come from a single fp16 pass, good to
// ~5e-4 / sqrt(Nt) of Nt: amp <= 0.06 sqrt(Nt) (R > 0.26 Nt at Nt = 512).  (ii) Where the sums are COHERENT -- f T < ~1, aliases of
// regular sampling, and above all series with a trend, whose low-frequency power is the largest on the grid -- the tensor core's
// round-toward-zero accumulation is a bias that the compensation model (tc_trunc_comp) removes only in part; measured on series
// with a drift of 1 ... 3 sigma over the span (refinement off, error in units of max P): <= 5e-5 below R = 0.6 Nt and 1.4e-4 above
// for the short-grid and batch kernels (2,048-sample drain windows); <= 4e-5 ... 9.5e-5 below R = 0.45 Nt and 1.5e-4 ... 2e-4 above
// for the CTA-pair kernel (4,096-sample windows); with long forced splits the short-grid kernel reached 8.8e-5 below 0.6 Nt too.
// Hence R > 0.45 Nt (amp 1.82) at the latest, for all of them.
// (In a periodogram of noise R / Nt ~ sqrt(ln Nf / Nt): 0.12 at Nt = 512.  Only f T < ~0.5 and aliases get there.)
__host__ __device__ inline double refine_amplification(bool tensor, int64_t Nt, bool gls = false, bool pair = false)
{
    if (!tensor) return 5.0;
    const double cap = 1.82; (void)pair;
    double a = 0.06 * sqrt((double)Nt);
    a = a < 1.35 ? 1.35 : (a > cap ? cap : a);
    if (!gls) return a;
    const double r = 1.0 - 1.0 / a;                                    // the same R / Nt, as a bound on the determinant
    return 1.0 / (1.0 - r * r);
}

// Tensor-core forms, strong lines: frequencies whose power exceeds refine_power() are refined as well.  Where the sums of a drain
// window are coherent AND the phases move slowly across it (time-sorted samples, f T (window / Nt) < ~1: a trend, a period comparable
// to the span), the products of an MMA come in two families, X cos a cos b and -X sin a sin b, whose signs are fixed over the window:
// the tensor core's per-product truncation then cancels between them or adds up, which the compensation model (tc_trunc_comp: sign
// excess from the window sum alone) cannot tell; and D_V, which has no compensation, loses in some windows and not in others.
// Measured (Nt = 1e5, drifts of 1 ... 100 sigma over the span, slow sinusoids and parabolas of 3 ... 30 sigma; refinement by R only):
// the error is a fraction of P_k ITSELF that saturates with the strength of the line -- CTA-pair kernel, 4,096-sample windows: 1.43e-4
// (1.58e-4 with fp16 lo planes), 7.7e-5 where the line holds 4 % of Nt, i.e. eps(P) ~ 1.43e-4 min(1, 2.8 sqrt(P / Nt)); 2,048-sample
// windows: 1.0e-4; short-grid kernel <= 5e-5, batch kernel <= 1.2e-5 at any strength.  Bins that are not refined are to stay within
// 4e-5 of THEIR OWN power (max P is at least that): P_k > 0.0118 Nt is refined -- with it the CTA-pair kernel measures <= 1e-5 of
// max P on all of those inputs.  Windows below 1,024 samples (32-sample splits of the short-grid kernel: C1, C2; short series) lose
// less: the threshold rises with (1,024 / window)^2 and soon passes (Nt - 1)/2, the largest power there is.  On noise next to nothing
// qualifies (P ~ Exp(1) against 0.0118 Nt: ~30 of C4's 8e6 bins, none from Nt = 2,048 on); a line of 20 % of the largest possible
// power (C3) has its main lobe refined: tens of bins.  The FP32-pipe form has no such term (INFINITY).  Applied by finish_kernel (the
// CTA-pair and short-grid kernels, batches with time splits); the fused epilogues of the batch kernel and of the shared-time GEMM do not
// test for it: those kernels measure <= 1.2e-5 and <= 1.5e-5 on the same inputs at any strength (one window of <= 2,048 samples per
// series there), and the test inside the epilogue's pipelined loop cost the shared-time GEMM half its speed at C4S.
__host__ __device__ inline float refine_power(bool tensor, int64_t Nt, int64_t window_samples)
{
    if (!tensor || window_samples <= 0) return INFINITY;
    const double s = window_samples >= 1024 ? 1.0 : 1024.0 / (double)window_samples;
    return (float)(0.0118 * (double)Nt * s * s);
}

constexpr int REFINE_THREADS = 256;
constexpr int REFINE_LIST_CAP = 1 << 20;     // entries of the list (8 bytes each: 8 MiB, allocated at the first call that needs it); overflow keeps the fp32-sum value

struct RefineSrc {
    const double* t; int64_t t_stride;      // the call's own inputs (device)
    const float* x; int64_t x_stride;
    const float* w; int64_t w_stride;       // nullable
    double f_min, df;
    int64_t Nt;
};

constexpr int REFINE_SPLIT_ENTRIES = 256;   // refine_kernel: up to this many listed frequencies of long series are each spread over ...
constexpr int REFINE_MAX_SPLIT = 64;        // ... up to this many blocks (ranges of samples), REFINE_SPLIT_MIN samples or more each
constexpr int REFINE_SPLIT_MIN = 1024;      // (fp64 sincospi is slow on this part: 1,000 samples per block take ~1 us)
constexpr int REFINE_WARP_MAX_NT = 4096;   // refine_kernel: series no longer than this get a warp per listed frequency instead of a block

struct RefineList {
    unsigned* head;                          // [0] entries appended, [1] blocks of refine_kernel done; both 0 between calls
    int2* items;                             // [REFINE_LIST_CAP] {series, frequency index}
    double* partial;                         // [REFINE_SPLIT_ENTRIES][REFINE_MAX_SPLIT][4] sums of a range of samples
    unsigned* entry_done;                    // [REFINE_SPLIT_ENTRIES] ranges of the entry summed so far; 0 between calls
};

__device__ __forceinline__ bool needs_refine(double CCh, double CS, double C1, double S1, double Nt, bool gls, double amp)
{
    if (gls) {
        const double cm = C1 / Nt, sm = S1 / Nt;
        const double CCn = 0.5 + CCh / Nt - cm * cm, SSn = 0.5 - CCh / Nt - sm * sm, CSn = CS / Nt - cm * sm;
        return !((CCn * SSn - CSn * CSn) * amp > 0.25);
    }
    const double thr = (1.0 - 1.0 / amp) * Nt;                         // R > thr
    return !(4.0 * (CCh * CCh + CS * CS) < thr * thr);
}

// false: the list is full (the caller keeps its own value and lets it take part in the arg-max)
__device__ __forceinline__ bool refine_push(const RefineList& L, int64_t b, int64_t k)
{
    const unsigned i = atomicAdd(L.head, 1u);
    if (i >= (unsigned)REFINE_LIST_CAP) return false;
    L.items[i] = make_int2((int)b, (int)k);
    return true;
}

// Sum over the block of NV values per thread, the same result in every thread: xor-butterfly inside a warp (both partners
// add the same two numbers), then the warps' sums in warp order.  `red` holds (NT / 32) * NV doubles.
// NT = 32: the team is ONE WARP of a larger block (short series: a warp per frequency); no shared memory, no barrier.
template <int NT, int NV>
__device__ __forceinline__ void refine_block_sum(double (&v)[NV], double* red)
{
    #pragma unroll
    for (int q = 0; q < NV; ++q)
        #pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    if (NT == 32) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();                                                    // (red may still be read from the previous call)
    if (lane == 0) {
        #pragma unroll
        for (int q = 0; q < NV; ++q) red[wid * NV + q] = v[q];
    }
    __syncthreads();
    #pragma unroll
    for (int q = 0; q < NV; ++q) {
        double a = 0.0;
        #pragma unroll
        for (int i = 0; i < NT / 32; ++i) a += red[i * NV + q];
        v[q] = a;
    }
}

// eq. (8) over the samples j0 <= j < j1 of series b at frequency k, in fp64: v = {XC, XS, CC - n/2, CS} (v[4], v[5] untouched = 0);
// `mean` = the (weighted) mean of x, `wn` = Nt / sum of the weights.  Time origin t_0: legal by eq. (2), keeps f t small.
template <int NT>
__device__ void refine_sums_range(const RefineSrc& s, int64_t b, int64_t k, double mean, double wn, int64_t j0, int64_t j1,
                                  double (&v)[6], double* red)
{
    const double* t = s.t + b * s.t_stride;
    const float* x = s.x + b * s.x_stride;
    const float* w = s.w ? s.w + b * s.w_stride : nullptr;
    const double t0 = __ldg(t), f = s.f_min + (double)k * s.df;
    for (int64_t j = j0 + (NT == 32 ? (threadIdx.x & 31) : threadIdx.x); j < j1; j += NT) {
        double ph = (__ldg(t + j) - t0) * f;
        ph -= rint(ph);
        double sn, cs;
        sincospi(2.0 * ph, &sn, &cs);
        const double wj = w ? wn * (double)__ldg(w + j) : 1.0;
        const double d = wj * ((double)__ldg(x + j) - mean);
        v[0] += d * cs; v[1] += d * sn;
        v[2] += wj * (cs * cs - 0.5); v[3] += wj * (cs * sn);
    }
    refine_block_sum<NT, 6>(v, red);
}

// The sums of frequency k of series b in fp64 (every thread of the block calls this with the same arguments and gets the same
// result), with the (weighted) mean removed from x and the weights scaled to mean 1:
//   eq. (8):            out = {XC, XS, CC - Nt/2, CS, -, -}, times from t_0
//   generalised form:   out = {XC', XS', CC', CS', SS', -} over the CENTRED basis c' = cos - mean(cos), s' = sin - mean(sin), times
//                       from their weighted mean: the fit is the same (the constant absorbs the means, the origin is free by eq. (2)),
//                       but CC' = sum w c'^2 is summed directly instead of CC - C^2/N, so nothing cancels as f T -> 0
//                       (cos - 1 = -2 sin^2 of the half angle: exact to fp64 relative precision however small)
template <int NT>
__device__ void refine_sums(const RefineSrc& s, int64_t b, int64_t k, bool gls, double (&out)[6], double* red /* (NT / 32) * 6 doubles */)
{
    const double* t = s.t + b * s.t_stride;
    const float* x = s.x + b * s.x_stride;
    const float* w = s.w ? s.w + b * s.w_stride : nullptr;
    const int64_t Nt = s.Nt;
    const int tid = NT == 32 ? (threadIdx.x & 31) : threadIdx.x;        // (NT = 32: a warp of a larger block)
    const double t0 = __ldg(t);
    double m[3] = {0.0, 0.0, 0.0};                                      // sum w, sum w x, sum w (t - t_0)
    for (int64_t j = tid; j < Nt; j += NT) {
        const double wj = w ? (double)__ldg(w + j) : 1.0;
        m[0] += wj; m[1] += wj * (double)__ldg(x + j); m[2] += wj * (__ldg(t + j) - t0);
    }
    refine_block_sum<NT, 3>(m, red);
    const double mean = m[1] / m[0], wn = (double)Nt / m[0];
    const double f = s.f_min + (double)k * s.df;
    double v[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (!gls) {
        refine_sums_range<NT>(s, b, k, mean, wn, 0, Nt, v, red);
    } else {
        const double tc = t0 + m[2] / m[0];                             // weighted mean time
        double a[2] = {0.0, 0.0};                                       // sum w (cos - 1), sum w sin
        for (int64_t j = tid; j < Nt; j += NT) {
            double ph = (__ldg(t + j) - tc) * f;
            ph -= rint(ph);
            double sh, ch;
            sincospi(ph, &sh, &ch);                                     // half angle
            const double wj = w ? wn * (double)__ldg(w + j) : 1.0;
            a[0] += wj * (-2.0 * sh * sh); a[1] += wj * (2.0 * sh * ch);
        }
        refine_block_sum<NT, 2>(a, red);
        const double cbar = a[0] / (double)Nt, sbar = a[1] / (double)Nt;   // (sum of the scaled weights = Nt)
        for (int64_t j = tid; j < Nt; j += NT) {
            double ph = (__ldg(t + j) - tc) * f;
            ph -= rint(ph);
            double sh, ch;
            sincospi(ph, &sh, &ch);
            const double wj = w ? wn * (double)__ldg(w + j) : 1.0;
            const double d = wj * ((double)__ldg(x + j) - mean);
            const double c1 = -2.0 * sh * sh - cbar, s1 = 2.0 * sh * ch - sbar;
            v[0] += d * c1; v[1] += d * s1;
            v[2] += wj * c1 * c1; v[3] += wj * c1 * s1; v[4] += wj * s1 * s1;
        }
        refine_block_sum<NT, 6>(v, red);
    }
    #pragma unroll
    for (int q = 0; q < 6; ++q) out[q] = v[q];
}

// Step 6 from fp64 sums: eq. (5) term by term; the second term is dropped where its denominator (Nt - R)/2 <= 1e-12 Nt,
// the oracle's own threshold for reading G7 (with fp32 sums finish_combine has to take 1e-6).  Generalised form: the
// Zechmeister-Kuerster quotient over the centred sums; singular (0, reading G7) where a basis function vanishes on the
// samples or the two coincide to 1e-12, as in the oracle's scaled elimination.
__device__ __forceinline__ double refine_combine(const double (&v)[6], double Nt, double inv2var, bool gls)
{
    const double XC = v[0], XS = v[1];
    if (gls) {
        const double CCn = v[2] / Nt, CSn = v[3] / Nt, SSn = v[4] / Nt;
        const double prod = CCn * SSn, D = prod - CSn * CSn;
        if (!(prod > 0.0) || !(D > 1e-12 * prod)) return 0.0;
        return fmax(SSn * XC * XC + CCn * XS * XS - 2.0 * CSn * XC * XS, 0.0) / (Nt * D) * inv2var;
    }
    const double CCh = v[2], CS = v[3];
    const double A = 2.0 * CCh, Bv = 2.0 * CS;
    const double R = sqrt(A * A + Bv * Bv);
    const double xc2 = XC * XC, xs2 = XS * XS, S = xc2 + xs2;
    const double D = R > 0.0 ? ((xc2 - xs2) * A + 2.0 * XC * XS * Bv) / R : 0.0;
    double val = fmax(S + D, 0.0) / (Nt + R);
    if (Nt - R > 2e-12 * Nt) val += fmax(S - D, 0.0) / (Nt - R);
    return val * inv2var;
}

struct RefineParams {
    RefineSrc src;
    RefineList list;
    const double* part_var; int nparts;     // [B][nparts]
    const double* part_sum;                  // [B][nparts] sum x (weighted: sum w x) from moments_kernel, or NULL: no spreading over blocks
    const double* part_w;                    // [B][nparts] sum w (weighted form), else NULL
    float* P; int64_t p_stride;              // nullable
    int32_t* peak_idx; float* peak_val; u64* peak64;   // nullable (all or none)
    int gls;
};

// Works off the list the fused epilogues left: grid-stride over its entries, one block per entry; the last block to finish
// publishes the peaks of the series it touched again and clears the list's head for the next call.
// grid: any (REFINE_GRID blocks), REFINE_THREADS threads.
__global__ void __launch_bounds__(REFINE_THREADS) refine_kernel(const RefineParams p)
{
    __shared__ double red[(REFINE_THREADS / 32) * 6];
    __shared__ unsigned s_last;
    pdl_wait();
    const unsigned appended = *reinterpret_cast<volatile unsigned*>(p.list.head);
    const unsigned n = appended < (unsigned)REFINE_LIST_CAP ? appended : (unsigned)REFINE_LIST_CAP;
    // long series, few entries: each entry's samples are cut into S ranges, one block each (a block sums 256 samples of fp64
    // sincospi in ~600 cycles whatever its size: the only way to go faster is more SMs); the block that finishes an entry last adds
    // the S partial sums in range order, so the result does not depend on which block that is
    const int64_t Nt = p.src.Nt;
    unsigned S = 1;
    if (!p.gls && p.part_sum && n > 0 && n <= (unsigned)REFINE_SPLIT_ENTRIES) {
        const int64_t by_len = Nt / REFINE_SPLIT_MIN;
        S = gridDim.x / n;
        if ((int64_t)S > by_len) S = (unsigned)by_len;
        if (S > (unsigned)REFINE_MAX_SPLIT) S = (unsigned)REFINE_MAX_SPLIT;
        if (S < 1) S = 1;
    }
    if (S > 1) {
        const unsigned item = blockIdx.x;                               // n S <= gridDim.x items
        if (item < n * S) {
            const unsigned e = item / S, r = item % S;
            const int2 it = p.list.items[e];
            const int64_t b = it.x, k = it.y;
            double sx = 0.0, sw = 0.0;                                  // (every thread: nparts <= 128 loads from L2)
            for (int i = 0; i < p.nparts; ++i) { sx += p.part_sum[b * p.nparts + i]; if (p.part_w) sw += p.part_w[b * p.nparts + i]; }
            if (!p.part_w) sw = (double)Nt;
            int64_t len = (Nt + S - 1) / S;
            len = (len + REFINE_THREADS - 1) / REFINE_THREADS * REFINE_THREADS;
            const int64_t j0 = (int64_t)r * len, j1 = (j0 + len < Nt) ? j0 + len : Nt;
            double v[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            refine_sums_range<REFINE_THREADS>(p.src, b, k, sx / sw, (double)Nt / sw, j0, j1, v, red);
            if (threadIdx.x == 0) {
                double* mine = p.list.partial + ((size_t)e * REFINE_MAX_SPLIT + r) * 4;
                mine[0] = v[0]; mine[1] = v[1]; mine[2] = v[2]; mine[3] = v[3];
                __threadfence();
                if (atomicAdd(p.list.entry_done + e, 1u) == S - 1) {    // the entry's last range: fold in range order
                    __threadfence();
                    double a[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
                    for (unsigned q = 0; q < S; ++q) {
                        const volatile double* part = p.list.partial + ((size_t)e * REFINE_MAX_SPLIT + q) * 4;
                        a[0] += part[0]; a[1] += part[1]; a[2] += part[2]; a[3] += part[3];
                    }
                    double qv = 0.0;
                    for (int i = 0; i < p.nparts; ++i) qv += p.part_var[b * p.nparts + i];
                    const float Pf = (float)refine_combine(a, (double)Nt, 0.5 / (qv / (double)(Nt - 1)), false);
                    if (p.P) p.P[b * p.p_stride + k] = Pf;
                    if (p.peak_idx) atomicMax(p.peak64 + b, ((u64)__float_as_uint(fmaxf(Pf, 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k));
                    p.list.entry_done[e] = 0u;                          // (for the next call)
                }
            }
        }
    } else if (Nt <= REFINE_WARP_MAX_NT) {
        // short series: a warp per entry (eight at a time per block); a block per entry would spend its time in the reductions
        const unsigned lane = threadIdx.x & 31u;
        for (unsigned e = blockIdx.x * (REFINE_THREADS / 32) + (threadIdx.x >> 5); e < n; e += gridDim.x * (REFINE_THREADS / 32)) {
            const int2 it = p.list.items[e];
            const int64_t b = it.x, k = it.y;
            double v[6];
            refine_sums<32>(p.src, b, k, p.gls != 0, v, nullptr);
            if (lane == 0) {
                double q = 0.0;
                for (int i = 0; i < p.nparts; ++i) q += p.part_var[b * p.nparts + i];
                const float Pf = (float)refine_combine(v, (double)Nt, 0.5 / (q / (double)(Nt - 1)), p.gls != 0);
                if (p.P) p.P[b * p.p_stride + k] = Pf;
                if (p.peak_idx) atomicMax(p.peak64 + b, ((u64)__float_as_uint(fmaxf(Pf, 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k));
            }
        }
    } else
    for (unsigned e = blockIdx.x; e < n; e += gridDim.x) {
        const int2 it = p.list.items[e];
        const int64_t b = it.x, k = it.y;
        double v[6];
        refine_sums<REFINE_THREADS>(p.src, b, k, p.gls != 0, v, red);
        if (threadIdx.x == 0) {
            double q = 0.0;
            for (int i = 0; i < p.nparts; ++i) q += p.part_var[b * p.nparts + i];
            const double var = q / (double)(p.src.Nt - 1);
            const float Pf = (float)refine_combine(v, (double)p.src.Nt, 0.5 / var, p.gls != 0);
            if (p.P) p.P[b * p.p_stride + k] = Pf;
            if (p.peak_idx) atomicMax(p.peak64 + b, ((u64)__float_as_uint(fmaxf(Pf, 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k));
        }
    }
    if (n == 0 && appended == 0) return;                                // nothing was flagged: head[1] stays 0
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = (atomicAdd(p.list.head + 1, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (p.peak_idx)
        for (unsigned e = threadIdx.x; e < n; e += REFINE_THREADS) {   // (several entries of one series write the same values)
            const int b = p.list.items[e].x;
            const u64 fin = *reinterpret_cast<volatile u64*>(p.peak64 + b);
            p.peak_idx[b] = (int32_t)(0xffffffffu - (unsigned)(fin & 0xffffffffull));
            p.peak_val[b] = __uint_as_float((unsigned)(fin >> 32));
        }
    __syncthreads();
    if (threadIdx.x == 0) { p.list.head[0] = 0u; p.list.head[1] = 0u; }
}

}  // namespace lsp
