// lsp_accum.cuh -- steps 3-5 of the hot path: anchor, rotate-and-accumulate, cascade.
//
// What it computes: the four sums of eq. (8) (SS is never formed)
//     XC = sum_j X_j cos(w t_j), XS = sum_j X_j sin(w t_j), CC = sum_j cos^2(w t_j), CS = sum_j cos sin
// for every frequency of a block over one split of the time axis.  Essentially all of the
// O(Nt*Nf) work of eq. (4) is in `pair_body`.
//
// How it differs from the paper's kernel (listing PAPER.md:138-277: one thread per frequency, one
// SFU sincos per term):
//   * each thread owns K ADJACENT frequencies k0..k0+K-1; for a sample j the angle at k0 is
//     evaluated once (32-bit fixed-point phase -> MUFU sin/cos) and then ADVANCED
//     K-1 times by the per-sample step 2 pi df t_j with a recurrence (the Press et al. idea the
//     paper sets aside at PAPER.md:59, made safe by re-anchoring every K steps);
//   * two consecutive samples ride in the two lanes of one packed f32x2 register, so every
//     instruction of the inner loop is an FFMA2 / FMUL2 doing two terms;
//   * chunked partial sums become: packed register partials per flush interval,
//     folded into per-thread shared-memory accumulators, written once per split to `ws`.
#pragma once
#include "lsp_common.cuh"

namespace lsp {

struct AccumParams {
    const float4* recA;
    const ulonglong2* recB;
    float* ws;              // [B][nsplit][4][Nf]
    int64_t Nt, Nf;
    int64_t split_len;      // samples per split (multiple of TILE; the last split may be shorter)
    int nsplit;
    int nfb;                // frequency blocks per series: ceil(Nf / (K * blockDim.x))
    int flush_tiles;        // tiles between folds of the register partials
};

constexpr int REC_ROTATION = 1;   // (c,s) <- (c cd - s sd, s cd + c sd): 8 FP32 lane-ops per term
constexpr int REC_THREE_TERM = 2; // c_{m+1} = 2 cd c_m - c_{m-1}:          6 FP32 lane-ops per term

// 2 pi / 2^32: signed 32-bit phase (turns * 2^32) -> radians in [-pi, pi)
#define LSP_RAD_PER_PHASE 1.4629180792671596e-9f

// One pair of samples (both lanes) against the thread's K frequencies.
template <int K, int REC, bool MASK>
__device__ __forceinline__ void pair_body(const float4 Av, const float4 Bv, const uint4 Cv, const unsigned tid,
                                          u64 (&XC)[K], u64 (&XS)[K], u64 (&CC)[K], u64 (&CS)[K])
{
    // step 3: anchor.  phase(k0) = b + tid * frac(K v)  (mod 1), exact integer wrap (reading G3)
    const int ph0 = (int)(Cv.x + tid * Cv.z);
    const int ph1 = (int)(Cv.y + tid * Cv.w);
    const float a0 = (float)ph0 * LSP_RAD_PER_PHASE;
    const float a1 = (float)ph1 * LSP_RAD_PER_PHASE;
    float c0 = __cosf(a0), s0 = __sinf(a0);
    float c1 = __cosf(a1), s1 = __sinf(a1);
    if (MASK) { c1 = 0.f; s1 = 0.f; }                     // phantom partner of an odd tail sample
    u64 c = pack2(c0, c1), s = pack2(s0, s1);
    const u64 X = pack2(Av.x, Av.y);
    const u64 cd = pack2(Bv.x, Bv.y), sd = pack2(Bv.z, Bv.w);

    if (REC == REC_THREE_TERM) {
        const u64 g = pack2(Av.z, Av.w);                  // 2 cos d
        u64 cp = fma2(c, cd, mul2(s, sd));                // cos(a - d): one exact backward rotation
        u64 sp = fma2(s, cd, neg2(mul2(c, sd)));          // sin(a - d)
        #pragma unroll
        for (int m = 0; m < K; ++m) {
            XC[m] = fma2(X, c, XC[m]);                    // step 4: the four sums of eq. (8)
            XS[m] = fma2(X, s, XS[m]);
            CC[m] = fma2(c, c, CC[m]);
            CS[m] = fma2(c, s, CS[m]);
            if (m + 1 < K) {
                const u64 cn = fma2(g, c, neg2(cp));
                const u64 sn = fma2(g, s, neg2(sp));
                cp = c; sp = s; c = cn; s = sn;
            }
        }
    } else {
        #pragma unroll
        for (int m = 0; m < K; ++m) {
            XC[m] = fma2(X, c, XC[m]);
            XS[m] = fma2(X, s, XS[m]);
            CC[m] = fma2(c, c, CC[m]);
            CS[m] = fma2(c, s, CS[m]);
            if (m + 1 < K) {
                const u64 t1 = mul2(s, sd);
                const u64 t2 = mul2(c, sd);
                const u64 cn = fma2(c, cd, neg2(t1));
                const u64 sn = fma2(s, cd, t2);
                c = cn; s = sn;
            }
        }
    }
}

// grid.x = B * nsplit * nfb (frequency block fastest), blockDim.x = T (multiple of 32, <= 256).
// dynamic shared memory: 3 * PAIRS * 16 bytes (tile) + 4 * K * T * 4 bytes (per-thread outer sums).
template <int K, int REC>
__global__ void __launch_bounds__(256) accum_kernel(const AccumParams p)
{
    extern __shared__ float4 lsp_smem[];
    float4* tA = lsp_smem;                                // {X0, X1, g0, g1}
    float4* tB = tA + PAIRS;                              // {cd0, cd1, sd0, sd1}
    uint4*  tC = reinterpret_cast<uint4*>(tB + PAIRS);    // {b0, b1, w0, w1}
    float* outer = reinterpret_cast<float*>(tC + PAIRS);  // [4][K][T]

    const int T = blockDim.x;
    const unsigned tid = threadIdx.x;
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t b = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * K * T;               // first frequency index of this block
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const float4* recA = p.recA + b * p.Nt;
    const ulonglong2* recB = p.recB + b * p.Nt;

    #pragma unroll
    for (int i = 0; i < 4 * K; ++i) outer[i * T + tid] = 0.f;

    u64 XC[K], XS[K], CC[K], CS[K];
    int64_t j = j_begin;
    int tiles_since_flush = 0;
    bool fresh = true;

    while (j < j_end) {
        const int ns = (int)min((int64_t)TILE, j_end - j);     // samples in this tile
        const int np = (ns + 1) >> 1;                          // pairs (the last may hold a phantom)
        if (fresh) {
            // partial CC is centred: each lane starts at -(pairs in the flush interval)/2
            const int64_t left = (j_end - j + 1) >> 1;
            const float ip = (float)min((int64_t)p.flush_tiles * PAIRS, left);
            const u64 init = pack2(-0.5f * ip, -0.5f * ip);
            #pragma unroll
            for (int m = 0; m < K; ++m) { XC[m] = 0ull; XS[m] = 0ull; CS[m] = 0ull; CC[m] = init; }
            fresh = false;
        }
        __syncthreads();                                       // previous tile fully consumed
        for (int i = tid; i < 2 * np; i += T) {
            float X = 0.f, cd = 1.f, sd = 0.f, g = 2.f;
            unsigned b32 = 0u, w32 = 0u;
            if (i < ns) {
                const float4 a = __ldg(recA + j + i);
                const ulonglong2 r = __ldg(recB + j + i);
                X = a.x; cd = a.y; sd = a.z; g = a.w;
                const u64 ph = r.x + (u64)kb * r.y;            // u + kb v  (mod 1, 64-bit wrap)
                b32 = (unsigned)((ph + 0x80000000ull) >> 32);
                w32 = (unsigned)(((u64)K * r.y + 0x80000000ull) >> 32);
            }
            const int pr = i >> 1, ln = i & 1;
            float* fa = reinterpret_cast<float*>(tA + pr);
            float* fbp = reinterpret_cast<float*>(tB + pr);
            unsigned* uc = reinterpret_cast<unsigned*>(tC + pr);
            fa[ln] = X;   fa[2 + ln] = g;
            fbp[ln] = cd; fbp[2 + ln] = sd;
            uc[ln] = b32; uc[2 + ln] = w32;
        }
        __syncthreads();

        const int nfull = (ns & 1) ? np - 1 : np;
        #pragma unroll 1
        for (int q = 0; q < nfull; ++q)
            pair_body<K, REC, false>(tA[q], tB[q], tC[q], tid, XC, XS, CC, CS);
        if (ns & 1)
            pair_body<K, REC, true>(tA[np - 1], tB[np - 1], tC[np - 1], tid, XC, XS, CC, CS);

        j += ns;
        if (++tiles_since_flush == p.flush_tiles || j >= j_end) {
            // step 5: cascade: fold the packed partials into the outer sums
            #pragma unroll
            for (int m = 0; m < K; ++m) {
                outer[(0 * K + m) * T + tid] += sum2(XC[m]);
                outer[(1 * K + m) * T + tid] += sum2(XS[m]);
                outer[(2 * K + m) * T + tid] += sum2(CC[m]);
                outer[(3 * K + m) * T + tid] += sum2(CS[m]);
            }
            tiles_since_flush = 0;
            fresh = true;
        }
    }

    float* ws = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
    #pragma unroll
    for (int m = 0; m < K; ++m) {
        const int64_t k = kb + (int64_t)tid * K + m;
        if (k < p.Nf) {
            ws[0 * p.Nf + k] = outer[(0 * K + m) * T + tid];
            ws[1 * p.Nf + k] = outer[(1 * K + m) * T + tid];
            ws[2 * p.Nf + k] = outer[(2 * K + m) * T + tid];
            ws[3 * p.Nf + k] = outer[(3 * K + m) * T + tid];
        }
    }
}

}  // namespace lsp
