// lsp_finish.cuh -- steps 6-7 of the hot path: combine the sums into P(f) and (optionally) the peak.
//
// Step 6 is eqs (5)-(7) with tau from eq. (6) eliminated algebraically, so no
// atan2 / sincos is needed (the listing calls atan2 + __sincosf):
//     A = CC - SS = 2 (CC - Nt/2),  B = 2 CS,  R = hypot(A, B)      [cos 2wtau = A/R, sin 2wtau = B/R]
//     S = XC^2 + XS^2,  D = ((XC^2 - XS^2) A + 2 XC XS B) / R
//     P = [ (S + D)/(Nt + R) + (S - D)/(Nt - R) ] / (2 var)  =  (S Nt - D R) / ((Nt^2 - R^2) var)
// (denominators of eq. (5) are (Nt +- R)/2, numerators (S +- D)/2).  All in fp64: O(Nf) work.
// Step 7: arg-max_k P with the lowest index among ties (reading G9), through one packed 64-bit
// atomicMax per block -- integer max is order-independent, so the result is deterministic.
#pragma once
#include "lsp_common.cuh"
#include "lsp_refine.cuh"

namespace lsp {

constexpr int FIN_THREADS = 256;

struct FinishParams {
    const float* ws;                   // [B][nsplit][4][Nf]
    const double* part_var;            // [B][nparts]
    float* P;                          // [B] x p_stride, nullable
    int64_t p_stride;
    int32_t* peak_idx;                 // [B], nullable
    float* peak_val;                   // [B], nullable
    u64* peak64;                       // [B]
    unsigned* counter;                 // [B]
    int64_t Nt, Nf;
    int nsplit, nparts;
    int x_scaled;                      // 1: XC, XS were accumulated from X * x_scale() (tensor-core forms)
    const float* ws1;                  // generalised periodogram: [B][nsplit][4][Nf] of the unit-weight pass (planes 0, 1 = sum cos, sum sin); else NULL
    const float* ws_x;                 // shared-time batch (lsp_shared_gemm.cuh): XC, XS from [B][nsplit][2][x_row]; `ws` is then ONE
    int64_t x_row;                     //   [nsplit][4][Nf] block shared by all series (planes 2, 3 = CC - n/2, CS); else NULL / 0
    RefineSrc src;                     // the raw series, for the ill-conditioned frequencies (lsp_refine.cuh)
    double refine_amp;                 // refine where the sums' rounding is amplified by more than this (refine_amplification); 0: nowhere
    float refine_pow;                  // ... and where P exceeds this (refine_power: strong lines on the tensor forms); INFINITY: nowhere
    RefineList list;                   // head != NULL (long series): append the flagged frequencies here for refine_kernel (one block each,
                                       //   in parallel) instead of redoing them one after the other inside this block
};

// Step 6 for one frequency from the six sums (C1, S1 only for the generalised periodogram), in fp64.
__device__ __forceinline__ double finish_combine(double XC, double XS, double CCh, double CS, double C1, double S1,
                                                 double Nt, double inv2var, bool gls)
{
    if (gls) {
        // Generalised (floating-mean) periodogram of Zechmeister & Kuerster 2009 (named at PAPER.md:375); the series is
        // already (weighted-)mean-subtracted, so Y = 0 and YC = XC/N, YS = XS/N; with per-sample weights every sum carries the
        // weights normalised to mean 1 (lsp_prepass.cuh), which leaves the formulas unchanged:
        //   CCn = CC/N - (C/N)^2, SSn = SS/N - (S/N)^2, CSn = CS/N - C S/N^2, D = CCn SSn - CSn^2
        //   P = (SSn XC^2 + CCn XS^2 - 2 CSn XC XS) / (2 var N D)        [same normalisation as eq. (1)]
        const double cm = C1 / Nt, sm = S1 / Nt;
        const double CCn = 0.5 + CCh / Nt - cm * cm, SSn = 0.5 - CCh / Nt - sm * sm, CSn = CS / Nt - cm * sm;
        const double D = CCn * SSn - CSn * CSn;
        if (!(D > 1e-9)) return 0.0;                                    // singular fit (f -> 0): 0, reading G7
        return fmax(SSn * XC * XC + CCn * XS * XS - 2.0 * CSn * XC * XS, 0.0) / (Nt * D) * inv2var;
    }
    // The two terms of eq. (5) over the common denominator (Nt + R)(Nt - R) = Nt^2 - R^2: one fp64 division, no square root:
    //   P 2 var = (S + D)/(Nt + R) + (S - D)/(Nt - R) = 2 (S Nt - D R) / (Nt^2 - R^2),   D R = (XC^2 - XS^2) A + 2 XC XS B
    const double A = 2.0 * CCh, Bv = 2.0 * CS;
    const double R2 = A * A + Bv * Bv;
    const double xc2 = XC * XC, xs2 = XS * XS;
    const double S = xc2 + xs2;
    const double DR = (xc2 - xs2) * A + 2.0 * XC * XS * Bv;
    double val;
    if (R2 < (1.0 - 1e-6) * (1.0 - 1e-6) * Nt * Nt) {
        val = fmax(2.0 * (S * Nt - DR), 0.0) / (Nt * Nt - R2);
    } else {                                                            // Nt - R <= 1e-6 Nt: the 0/0 term is dropped (reading G7)
        const double R = sqrt(R2);
        val = fmax(S + DR / R, 0.0) / (Nt + R);
    }
    return val * inv2var;
}

// grid (ceil(Nf / FIN_BLOCK_F), B), FIN_THREADS threads = FIN_SL split lanes x FIN_BLOCK_F frequencies: thread (l, f) sums
// the time splits sp = l, l + FIN_SL, ... of frequency f in that order (independent loads, all in flight at once); the
// FIN_SL partial sums are then added in lane order by the l = 0 thread.  The order is fixed, so the result is
// deterministic; with few frequencies and many splits (C1, C2) the sum over the splits is no longer one long dependent chain.
// FIN_SL = 1 (few splits): one thread per frequency, 256 frequencies per block, no exchange.
// Frequencies whose sums are ill-conditioned (needs_refine) are then redone by the whole block in fp64, one after the other.
template <int FIN_SL, bool LOOP>
__global__ void __launch_bounds__(FIN_THREADS) finish_kernel(const FinishParams p)
{
    constexpr int FIN_BLOCK_F = FIN_THREADS / FIN_SL;
    __shared__ double s_var, s_var_raw;
    __shared__ int s_nflag;
    __shared__ short s_flag[FIN_BLOCK_F];
    __shared__ double s_red[(FIN_THREADS / 32) * 6];
    __shared__ double s_part[FIN_SL > 1 ? 6 : 1][FIN_SL][FIN_SL > 1 ? FIN_BLOCK_F : 1];
    __shared__ u64 s_best[FIN_THREADS / 32];
    const int64_t b = blockIdx.y;
    const int fl = threadIdx.x % FIN_BLOCK_F, sl = threadIdx.x / FIN_BLOCK_F;
    pdl_wait();                                            // (launched as a programmatic dependent of the accumulate kernel on the short-grid path)
    if (threadIdx.x == 0) {
        double q = 0.0;                                    // fixed-order sum of the block partials
        for (int i = 0; i < p.nparts; ++i) q += p.part_var[b * p.nparts + i];
        s_var = q / (double)(p.Nt - 1);                    // sample variance (reading G1)
        s_var_raw = s_var;
        s_nflag = 0;
        if (p.x_scaled) {                                  // undo the fp32 scale factor exactly (lsp_tc.cuh)
            const double xs = (double)(float)(1.0 / sqrt(s_var));
            s_var *= xs * xs;
        }
    }
    const float* ws = p.ws_x ? p.ws : p.ws + b * p.nsplit * 4 * p.Nf;
    const float* wx = p.ws_x ? p.ws_x + b * p.nsplit * 2 * p.x_row : nullptr;
    const float* w1 = p.ws1 ? p.ws1 + b * p.nsplit * 4 * p.Nf : nullptr;
    const bool gls = p.ws1 != nullptr;
    const int64_t nchunk = (p.Nf + FIN_BLOCK_F - 1) / FIN_BLOCK_F;
    u64 best = 0ull;

    // LOOP (batches): a block takes the chunks blockIdx.x, blockIdx.x + gridDim.x, ... of its series -- a batch of short grids would
    // otherwise be tens of thousands of blocks that each pay the serial prologue above (0.19 -> 0.13 ms at C4).  Otherwise one chunk
    // per block, straight-line code (gridDim.x = nchunk).
    int64_t c = blockIdx.x;
    do {
        const int64_t k = c * FIN_BLOCK_F + fl;
        const bool live = k < p.Nf;

        double XC = 0.0, XS = 0.0, CCh = 0.0, CS = 0.0, C1 = 0.0, S1 = 0.0;
        if (live) {
            #pragma unroll 2
            for (int sp = sl; sp < p.nsplit; sp += FIN_SL) {   // fixed order over this lane's time splits
                const float* w = ws + (int64_t)sp * 4 * p.Nf + k;
                if (wx) {
                    XC += (double)__ldg(wx + (int64_t)sp * 2 * p.x_row + k);
                    XS += (double)__ldg(wx + (int64_t)sp * 2 * p.x_row + p.x_row + k);
                } else {
                    XC += (double)__ldg(w);
                    XS += (double)__ldg(w + p.Nf);
                }
                CCh += (double)__ldg(w + 2 * p.Nf);
                CS += (double)__ldg(w + 3 * p.Nf);
                if (w1) {
                    C1 += (double)__ldg(w1 + (int64_t)sp * 4 * p.Nf + k);
                    S1 += (double)__ldg(w1 + (int64_t)sp * 4 * p.Nf + p.Nf + k);
                }
            }
        }
        if (FIN_SL > 1) {
            s_part[0][sl][fl] = XC; s_part[1][sl][fl] = XS; s_part[2][sl][fl] = CCh; s_part[3][sl][fl] = CS;
            s_part[4][sl][fl] = C1; s_part[5][sl][fl] = S1;
        }
        __syncthreads();                                   // s_var, s_nflag (thread 0's prologue runs beside the loads above); the lanes' partial sums
        const bool owner = live && sl == 0;
        double v[6] = {XC, XS, CCh, CS, C1, S1};
        if (owner && FIN_SL > 1) {
            #pragma unroll
            for (int q = 0; q < 6; ++q) {
                double a = 0.0;
                #pragma unroll
                for (int l = 0; l < FIN_SL; ++l) a += s_part[q][l][fl];   // fixed order over the lanes
                v[q] = a;
            }
        }
        float Pf = 0.f;
        if (owner) Pf = (float)finish_combine(v[0], v[1], v[2], v[3], v[4], v[5], (double)p.Nt, 0.5 / s_var, gls);
        bool listed = false;                               // refine_kernel will write this frequency and enter it in the arg-max
        if (p.refine_amp > 0.0 && p.list.head) {
            if (owner && (needs_refine(v[2], v[3], v[4], v[5], (double)p.Nt, gls, p.refine_amp) || Pf > p.refine_pow)) listed = refine_push(p.list, b, k);
        } else if (p.refine_amp > 0.0) {                   // (uniform over the grid)
            if (owner && (needs_refine(v[2], v[3], v[4], v[5], (double)p.Nt, gls, p.refine_amp) || Pf > p.refine_pow)) s_flag[atomicAdd(&s_nflag, 1)] = (short)fl;
            __syncthreads();
            const int nflag = s_nflag;
            for (int i = 0; i < nflag; ++i) {              // the order of the list varies from run to run; each entry's result does not
                const int f = s_flag[i];
                double r[6];
                refine_sums<FIN_THREADS>(p.src, b, c * FIN_BLOCK_F + f, gls, r, s_red);
                if (owner && fl == f) Pf = (float)refine_combine(r, (double)p.Nt, 0.5 / s_var_raw, gls);
            }
        }
        if (owner) {
            if (p.P) p.P[b * p.p_stride + k] = Pf;
            if (!listed) {
                const u64 key = ((u64)__float_as_uint(fmaxf(Pf, 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k);
                best = (key > best) ? key : best;
            }
        }
        if (!LOOP) break;
        c += gridDim.x;
        if (c < nchunk) {                                  // another chunk follows (uniform): the shared arrays are free again after this
            __syncthreads();
            if (threadIdx.x == 0) s_nflag = 0;
        }
    } while (c < nchunk);
    if (p.peak_idx == nullptr || sl != 0) return;          // (whole warps: FIN_BLOCK_F is a multiple of 32)
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const u64 other = __shfl_down_sync(0xffffffffu, best, o);
        best = (other > best) ? other : best;
    }
    if (FIN_SL == 1) {                                     // eight warps: fold them through shared memory first
        if ((threadIdx.x & 31) == 0) s_best[threadIdx.x >> 5] = best;
        __syncthreads();
        if (threadIdx.x == 0) for (int i = 1; i < FIN_THREADS / 32; ++i) best = (s_best[i] > best) ? s_best[i] : best;
    }
    if (threadIdx.x == 0) {
        atomicMax(p.peak64 + b, best);
        __threadfence();
        const unsigned done = atomicAdd(p.counter + b, 1u);
        if (done == gridDim.x - 1) {                       // last block of this series: publish
            __threadfence();
            const u64 fin = atomicMax(p.peak64 + b, 0ull);
            p.peak_idx[b] = (int32_t)(0xffffffffu - (unsigned)(fin & 0xffffffffull));
            p.peak_val[b] = __uint_as_float((unsigned)(fin >> 32));
        }
    }
}

}  // namespace lsp
