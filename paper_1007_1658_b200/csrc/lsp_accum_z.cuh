// lsp_accum_z.cuh -- steps 3-5 of the hot path on the FP32 pipe: anchor, rotate-and-accumulate, cascade.
//
// What it computes: the four sums of eq. (8) (SS is never formed)
//     XC = sum_j X_j cos(w t_j), XS = sum_j X_j sin(w t_j), CC = sum_j cos^2(w t_j), CS = sum_j cos sin
// for every frequency of a block over one split of the time axis: all of the O(Nt*Nf) work of eq. (4)
// in the paper's own arithmetic (fp32 throughout, with the SFU for the trig).
//
// How it differs from the paper's kernel (listing PAPER.md:138-277: one thread per frequency, one SFU sincos per term):
//   * each thread owns K ADJACENT frequencies k0..k0+K-1; for a sample j the angle at k0 is evaluated once (32-bit
//     fixed-point phase -> MUFU sin/cos) and then ADVANCED K-1 times by the per-sample step 2 pi df t_j with the
//     three-term recurrence z_{m+1} = 2 cos(d) z_m - z_{m-1} (the Press et al. idea the paper sets aside at PAPER.md:59,
//     made safe by re-anchoring every K <= 32 steps from an exact integer phase);
//   * the two lanes of a packed f32x2 register hold z_m = (cos th_m, sin th_m), th_m = w_{k0+m} t_j.  Per term
//
//     (XC, XS)_m += X      * z_m        FFMA2  X.F32 (scalar broadcast), z, acc1
//     (CC, CS)_m += cos th * z_m        FFMA2  z.lo.F32 (scalar broadcast), z, acc2
//     z_{m+1}     = g * z_m - z_{m-1}   FFMA2  g.F32, z, -z_{m-1}          g = 2 cos(2 pi df t_j)
//
// = 3 packed instructions = 6 FP32 lane-ops per term.  Why this layout on sm_100a (measured, see
// DESIGN.md "Register-file model"): an FFMA2 issues every 2 cycles only if at most two of its
// 64-bit operands are fetched from the register file; here all three instructions of a term share
// the multiplicand z (operand-reuse cache) and the other multiplicand is a 32-bit scalar, so the
// limit is met whatever order ptxas picks.  The accumulators cost 4 registers per frequency,
// so K = 24..32 adjacent frequencies fit per thread and the MUFU anchor
// is amortised over many terms.  Chunked partial sums become: packed register partials per
// flush interval, folded into per-thread shared-memory accumulators, written once per split to `ws`.
#pragma once
#include "lsp_common.cuh"

namespace lsp {

struct AccumParams {
    const float4* recW;     // weighted generalised periodogram: recW[j].x = sqrt of the normalised weight (anchors are scaled by it); else NULL
    const float4* recA;
    const ulonglong2* recB;
    float* ws;              // [B][nsplit][4][Nf]
    float* ws1;             // GLS kernels: [B][nsplit][4][Nf], planes 0, 1 = sum (w) cos, sum (w) sin (the generalised periodogram's C, S)
    int64_t Nt, Nf;
    int64_t split_len;      // samples per split (multiple of TILE_Z; the last split may be shorter)
    int nsplit;
    int nfb;                // frequency blocks per series: ceil(Nf / (K * blockDim.x))
    int flush_tiles;        // tiles of TILE_Z samples between folds of the register partials
};

struct ZAnchor { float c0, s0, cp, sp, X, g, sw; };

// step 3: anchor at the thread's first frequency: exact integer phase (reading G3) -> MUFU sin/cos
// (PAPER.md:290), plus the value one recurrence step back by an exact rotation (consistent with the
// anchor, so the anchor's own error is not amplified by the three-term recurrence).
// WEIGHTED (weighted generalised periodogram): the tile also holds sw = sqrt(normalised weight) and the anchor pair is
// scaled by it: the recurrence is linear, so z_m = sw e^{i th_m} throughout and, with X = sw x, the sums become
// sum w x e^{i th} and sum w cos th e^{i th} at no cost per term (4 more FMUL per sample).
template <bool WEIGHTED>
__device__ __forceinline__ ZAnchor z_anchor(const float4* tS, const void* tRv, int q, unsigned tid)
{
    const float4 sv = tS[q];
    float cd, sd, sw = 1.f;
    if (WEIGHTED) { const float4 rv = static_cast<const float4*>(tRv)[q]; cd = rv.x; sd = rv.y; sw = rv.z; }
    else { const float2 rv = static_cast<const float2*>(tRv)[q]; cd = rv.x; sd = rv.y; }
    const int ph = (int)(__float_as_uint(sv.z) + tid * __float_as_uint(sv.w));
    const float ang = (float)ph * LSP_RAD_PER_PHASE;
    ZAnchor a;
    a.c0 = __cosf(ang); a.s0 = __sinf(ang);
    if (WEIGHTED) { a.c0 *= sw; a.s0 *= sw; }
    a.cp = fmaf(a.c0, cd, a.s0 * sd);
    a.sp = fmaf(a.s0, cd, -(a.c0 * sd));
    a.X = sv.x; a.g = sv.y; a.sw = sw;
    return a;
}

// DIRECT (the CTA's whole time split fits ONE fold interval, e.g. batches of short series): the register partials are the
// split's sums and go straight to `ws`; no shared-memory accumulators, so more CTAs fit per SM (C4: 6 instead of 5).
// GLS (generalised periodogram in ONE pass: "two more FMAs per term in the same kernel"): a third packed
// accumulator per frequency, (C, S)_m += sw * z_m (sw = 1 without weights; with weights z carries one sqrt(w) already), one more
// FFMA2 per term = 8 lane-ops instead of the 12 of two passes; 2 K more registers, so K <= 20.
template <int K, int MAXT, int MINB, bool WEIGHTED = false, bool DIRECT = false, bool GLS = false>
__global__ void __launch_bounds__(MAXT, MINB) accum_z_kernel(const AccumParams p)
{
    constexpr int NQ = GLS ? 6 : 4;                            // sums per frequency
    extern __shared__ float4 lsp_smem[];
    float4* tS = lsp_smem;                                     // {X, g, b32, w32} per sample
    void* tR = tS + TILE_Z;                                    // {cd, sd} per sample (WEIGHTED: {cd, sd, sw, -}, the tile region is sized for it)
    float* outer = reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(tR) + TILE_Z * (WEIGHTED ? 16 : 8));   // [T][4K+1] (odd stride: conflict-free)

    const int T = blockDim.x;
    const unsigned tid = threadIdx.x;
#ifndef LSP_Z_OUTER_TM
#define LSP_Z_OUTER_TM 1
#endif
#if LSP_Z_OUTER_TM
#define OIDX(q, m) (tid * (NQ * K + 1) + (q) * K + (m))
#else
#define OIDX(q, m) (((q) * K + (m)) * T + tid)
#endif
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t b = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * K * T;                    // first frequency index of this block
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const float4* recA = p.recA + b * p.Nt;
    const ulonglong2* recB = p.recB + b * p.Nt;
    const int flush_tiles = DIRECT ? 0x7fffffff / TILE_Z : max(1, p.flush_tiles);

    if (!DIRECT) {
        #pragma unroll
        for (int i = 0; i < NQ * K; ++i) outer[OIDX(i / K, i % K)] = 0.f;
    }

    u64 A1[K], A2[K];                                          // (XC, XS), (CC - n/2, CS)
    u64 A3[GLS ? K : 1];                                       // GLS: (C, S)
    int64_t j = j_begin;
    int tiles_since_flush = 0;
    bool fresh = true;
    if (DIRECT) {                                              // one interval: the whole split
        const u64 init = pack2(-0.5f * (float)max((int64_t)0, j_end - j_begin), 0.f);
        #pragma unroll
        for (int m = 0; m < K; ++m) { A1[m] = 0ull; A2[m] = init; if (GLS) A3[m] = 0ull; }
        fresh = false;
    }

    while (j < j_end) {
        const int ns = (int)min((int64_t)TILE_Z, j_end - j);
        if (fresh) {
            const float n_int = (float)min((int64_t)flush_tiles * TILE_Z, j_end - j);
            const u64 init = pack2(-0.5f * n_int, 0.f);        // centred CC partial
            #pragma unroll
            for (int m = 0; m < K; ++m) { A1[m] = 0ull; A2[m] = init; if (GLS) A3[m] = 0ull; }
            fresh = false;
        }
        __syncthreads();                                       // previous tile fully consumed
        for (int i = tid; i < ns; i += T) {
            const float4 a = __ldg(recA + j + i);
            const ulonglong2 r = __ldg(recB + j + i);
            const u64 ph = r.x + (u64)kb * r.y;                // u + kb v  (mod 1, 64-bit wrap)
            const unsigned b32 = (unsigned)((ph + 0x80000000ull) >> 32);
            const unsigned w32 = (unsigned)(((u64)K * r.y + 0x80000000ull) >> 32);
            tS[i] = make_float4(a.x, a.w, __uint_as_float(b32), __uint_as_float(w32));
            if (WEIGHTED) static_cast<float4*>(tR)[i] = make_float4(a.y, a.z, __ldg(&p.recW[b * p.Nt + j + i].x), 0.f);
            else static_cast<float2*>(tR)[i] = make_float2(a.y, a.z);
        }
        __syncthreads();

        // Software pipeline: the anchor of sample q+1 (LDS -> IMAD -> I2F -> MUFU, ~100 cycles of
        // dependent latency) is issued under the FFMA2 stream of sample q.
#ifndef LSP_Z_PIPE
#define LSP_Z_PIPE 0
#endif
#if LSP_Z_PIPE
        ZAnchor nx = z_anchor<WEIGHTED>(tS, tR, 0, tid);
#endif
        #pragma unroll 1
        for (int q = 0; q < ns; ++q) {
#if LSP_Z_PIPE
            const ZAnchor cur = nx;
            nx = z_anchor<WEIGHTED>(tS, tR, min(q + 1, ns - 1), tid);
#else
            const ZAnchor cur = z_anchor<WEIGHTED>(tS, tR, q, tid);
#endif
            u64 z = pack2(cur.c0, cur.s0);
            u64 zp = pack2(cur.cp, cur.sp);
            const u64 XX = pack2(cur.X, cur.X), GG = pack2(cur.g, cur.g);
            const u64 SW = pack2(cur.sw, cur.sw);              // (GLS only)
            // step 4
            #pragma unroll
            for (int m = 0; m < K; ++m) {
                float cm, sm; unpack2(z, cm, sm);
                A1[m] = fma2(XX, z, A1[m]);
                A2[m] = fma2(pack2(cm, cm), z, A2[m]);
                if (GLS) A3[m] = fma2(SW, z, A3[m]);
                if (m + 1 < K) { const u64 zn = fma2(GG, z, neg2(zp)); zp = z; z = zn; }
            }
        }

        j += ns;
        if (!DIRECT && (++tiles_since_flush == flush_tiles || j >= j_end)) {
            // step 5: cascade
            #pragma unroll
            for (int m = 0; m < K; ++m) {
                float xc, xs, cc, cs;
                unpack2(A1[m], xc, xs); unpack2(A2[m], cc, cs);
                outer[OIDX(0, m)] += xc;
                outer[OIDX(1, m)] += xs;
                outer[OIDX(2, m)] += cc;
                outer[OIDX(3, m)] += cs;
                if (GLS) { float c1, s1; unpack2(A3[m], c1, s1); outer[OIDX(4, m)] += c1; outer[OIDX(5, m)] += s1; }
            }
            tiles_since_flush = 0;
            fresh = true;
        }
    }

    float* ws = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
    float* ws1 = GLS ? p.ws1 + ((b * p.nsplit + sp) * 4) * p.Nf : nullptr;
    #pragma unroll
    for (int m = 0; m < K; ++m) {
        const int64_t k = kb + (int64_t)tid * K + m;
        if (k < p.Nf) {
            if (GLS) {
                if (DIRECT) { float c1, s1; unpack2(A3[m], c1, s1); ws1[k] = c1; ws1[p.Nf + k] = s1; }
                else { ws1[k] = outer[OIDX(4, m)]; ws1[p.Nf + k] = outer[OIDX(5, m)]; }
            }
            if (DIRECT) {
                float xc, xs, cc, cs;
                unpack2(A1[m], xc, xs); unpack2(A2[m], cc, cs);
                ws[0 * p.Nf + k] = xc; ws[1 * p.Nf + k] = xs; ws[2 * p.Nf + k] = cc; ws[3 * p.Nf + k] = cs;
            } else {
            ws[0 * p.Nf + k] = outer[OIDX(0, m)];
            ws[1 * p.Nf + k] = outer[OIDX(1, m)];
            ws[2 * p.Nf + k] = outer[OIDX(2, m)];
            ws[3 * p.Nf + k] = outer[OIDX(3, m)];
            }
        }
    }
}

}  // namespace lsp
