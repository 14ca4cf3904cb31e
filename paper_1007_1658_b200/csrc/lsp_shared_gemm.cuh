// lsp_shared_gemm.cuh -- the shared-time batch: B series on ONE set of sample times.
//
// This is the Monte-Carlo use the paper describes: keep the sampling, redraw the noise, take the peak
// of each periodogram.  With the times shared, the trig factors of eq. (8) do not depend on the
// series, so
//     XC[b,k] = sum_j X_bj cos th_jk,   XS[b,k] = sum_j X_bj sin th_jk,   th_jk = 2 pi frac(u_j + k v_j)   (exact turns, G3)
// is a genuinely dense contraction  D[b][(k,part)] = sum_j X[b][j] E[(k,part)][j]  --  M = series, N = (frequency,
// cos | sin), K = samples -- and CC, CS (hence tau, eq. (2)) are computed ONCE per frequency instead of once per series.
//
// Pre-passes (all O(Nt (Nf + B))):
//   shared_e_kernel   E as tcgen05 B-operand tiles (no-swizzle K-major core matrices, fp16 plane + e5m2 plane), one
//                     MUFU sin/cos per (sample, frequency).
//   shared_v_kernel   CC - n/2, CS per frequency and time split (one warp each, fixed shuffle tree).
//   shared_x_kernel   X / sigma_b as A-operand tiles (fp16 plane + e5m2 plane).
// shared_gemm_kernel  a TMA-fed tcgen05 GEMM: CTA tile 128 series x 128 frequencies (N = 256) x one time split; one
//                     thread streams the pre-tiled operands with cp.async.bulk (48 KB per stage of 32 samples, 4 stages),
//                     one thread issues per 16 samples  D += X_hi E_hi (kind::f16)  and  D += [X_lo|X_hi8][E_hi8|E_lo]
//                     (kind::f8f6f4, e5m2: both first-order corrections in one MMA of K = 32), accumulators in 256 TMEM
//                     columns; 4 warps drain them to ws_x[b][split][part][k].  A time split is at most 2,048 samples, so the
//                     truncating tensor-core accumulation is folded as often as in the single-series forms.
#pragma once
#include "lsp_tc.cuh"
#include "lsp_refine.cuh"

namespace lsp {

constexpr int SG_KS = 16;                                  // samples per k-step (fp16 MMA K)
constexpr int SG_M = 128;                                  // series per CTA
constexpr int SG_F = 128;                                  // frequencies per CTA (N = 2 SG_F)
constexpr int SG_A_PLANE = SG_M * 32;                      // 4 KB: 128 rows x 16 samples fp16 (or 32 e5m2)
constexpr int SG_B_PLANE = 2 * SG_F * 32;                  // 8 KB
constexpr int SG_A_GROUP = 2 * SG_A_PLANE;                 // per k-step: fp16 plane + e5m2 plane
constexpr int SG_B_GROUP = 2 * SG_B_PLANE;
constexpr int SG_KPS = 2;                                  // k-steps per stage
constexpr int SG_STAGES = 2;                                 // x 48 KB: two CTAs per SM (256 TMEM columns each), so one CTA's epilogue overlaps the other's main loop
constexpr int SG_STAGE_BYTES = SG_KPS * (SG_A_GROUP + SG_B_GROUP);
constexpr size_t SG_SMEM = (size_t)SG_STAGES * SG_STAGE_BYTES + 256;
constexpr int SG_THREADS = 6 * 32;                         // warp 0: TMA, warp 1: MMA + TMEM, warps 2-5: drain
constexpr int SG_MAX_SPLIT = 2048;                         // samples per time split (multiple of SG_KPS * SG_KS)
constexpr int SG_TMEM_COLS = 256;
constexpr uint32_t SG_IDESC = umma_idesc(SG_M, 2 * SG_F);

struct SharedGemmParams {
    const unsigned char* xa;        // [nmb][ng][SG_A_GROUP]
    const unsigned char* eb;        // [nfb][ng][SG_B_GROUP]: the E tiles of ONE BAND of nfb frequency blocks starting at block nb0
    float* ws_x;                    // [B][nsplit][2][x_row]
    int64_t B, Nf, x_row;
    int nmb, nfb, nsplit, ng;       // ng = k-step groups over ALL splits = nsplit * groups_per_split; nfb = frequency blocks of this launch (band)
    int nb0, nfb_total;             // first frequency block of the band; blocks of the whole grid (the last one publishes the peak)
    int groups_per_split;           // even
    // fused steps 6-7 (only when nsplit == 1: the accumulators ARE the sums of eq. (8)); vconst == NULL: write ws_x instead
    const double* vconst;           // [4][Nf]: cos 2 w tau, sin 2 w tau, 1/(Nt + R), 1/(Nt - R) (0 if dropped, reading G7)
    const float4* vconst_f;         // [Nf]: the same four as fp32, .x = NaN where R > Nt/2 (the difference S - D is then formed in fp64)
    const double* part_var;         // [B][nparts]
    float* P; int64_t p_stride;     // nullable
    int32_t* peak_idx; float* peak_val; u64* peak64; unsigned* counter;   // nullable (all or none)
    int64_t Nt; int nparts;
    RefineList list;                // fused epilogue: where the ill-conditioned frequencies go (lsp_refine.cuh); head NULL: nowhere
    double refine_thr;              //   ... those with R > refine_thr Nt (refine_amplification)
};

// Per-frequency part of step 6 for the shared-time batch: from CC - n/2, CS (summed over the splits in fixed order)
// A = CC - SS, B = 2 CS, R = hypot(A, B) -> (A/R, B/R, 1/(Nt + R), 1/(Nt - R)); eqs (5)-(7), tau eliminated.
__global__ void __launch_bounds__(256) shared_vconst_kernel(const float* __restrict__ ws_v, int nsplit, int64_t Nf, int64_t Nt_i, double* __restrict__ vconst,
                                                            float4* __restrict__ vconst_f, double redo_thr /* <= 0.5: fp32 below R = redo_thr Nt */)
{
    pdl_trigger();                                          // (the kernels of a shared-time call are launched as programmatic dependents:
    pdl_wait();                                             //  launch and set-up overlap the predecessor's tail; nothing is read or written before this)
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= Nf) return;
    double CCh = 0.0, CS = 0.0;
    for (int sp = 0; sp < nsplit; ++sp) { CCh += (double)ws_v[((int64_t)sp * 4 + 2) * Nf + k]; CS += (double)ws_v[((int64_t)sp * 4 + 3) * Nf + k]; }
    const double Nt = (double)Nt_i, A = 2.0 * CCh, Bv = 2.0 * CS, R = hypot(A, Bv);
    vconst[k] = (R > 0.0) ? A / R : 0.0;
    vconst[Nf + k] = (R > 0.0) ? Bv / R : 0.0;
    vconst[2 * Nf + k] = 1.0 / (Nt + R);
    vconst[3 * Nf + k] = (Nt - R > 1e-6 * Nt) ? 1.0 / (Nt - R) : 0.0;
    // fp32 copy for the common case R <= Nt/2 (1/(Nt - R) <= 3/(Nt + R): no amplification of the fp32 rounding of S - D)
    vconst_f[k] = make_float4((R <= redo_thr * Nt) ? (float)vconst[k] : __int_as_float(0x7fc00000), (float)vconst[Nf + k],
                              (float)vconst[2 * Nf + k], (float)vconst[3 * Nf + k]);
}

// ------------------------------------------------------------------ E tiles + partial CC, CS
// grid (band blocks, ng), 256 threads: kf = tid & 127 (frequency k = 128 (nb0 + block) + kf), chunk = tid >> 7 (8 of the group's
// 16 samples).  E is made one BAND of frequency blocks at a time (the host bounds the buffer), block `nb` of the band at eb[nb].
__global__ void __launch_bounds__(256) shared_e_kernel(const ulonglong2* __restrict__ recB, int64_t Nt, int64_t Nf,
                                                       unsigned char* __restrict__ eb, int ng, int nb0)
{
    pdl_trigger();                                          // (the kernels of a shared-time call are launched as programmatic dependents:
    pdl_wait();                                             //  launch and set-up overlap the predecessor's tail; nothing is read or written before this)
    const int nb = blockIdx.x, g = blockIdx.y;
    const unsigned kf = threadIdx.x & 127u, chunk = threadIdx.x >> 7;
    const int64_t k = (int64_t)(nb0 + nb) * SG_F + kf;
    float c[8], s[8];
    #pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int64_t j = (int64_t)g * SG_KS + chunk * 8 + i;
        c[i] = 0.f; s[i] = 0.f;
        if (j < Nt && k < Nf) {
            const ulonglong2 r = __ldg(recB + j);
            const u64 ph = r.x + (u64)k * r.y;                          // u + k v (mod 1, exact 64-bit wrap; reading G3)
            sincos_phase32((unsigned)((ph + 0x80000000ull) >> 32), c[i], s[i]);
        }
    }
    unsigned ch[4], sh[4], c8h[2], s8h[2], c8l[2], s8l[2];
    #pragma unroll
    for (int i = 0; i < 4; ++i) { ch[i] = pack_h2(c[2 * i], c[2 * i + 1]); sh[i] = pack_h2(s[2 * i], s[2 * i + 1]); }
    #pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float2 a = unpack_h2(ch[2 * i]), b2 = unpack_h2(ch[2 * i + 1]);
        c8h[i] = pack_e5m2_h2(ch[2 * i]) | (pack_e5m2_h2(ch[2 * i + 1]) << 16);
        c8l[i] = pack_e5m2(c[4 * i] - a.x, c[4 * i + 1] - a.y) | (pack_e5m2(c[4 * i + 2] - b2.x, c[4 * i + 3] - b2.y) << 16);
        const float2 d = unpack_h2(sh[2 * i]), e = unpack_h2(sh[2 * i + 1]);
        s8h[i] = pack_e5m2_h2(sh[2 * i]) | (pack_e5m2_h2(sh[2 * i + 1]) << 16);
        s8l[i] = pack_e5m2(s[4 * i] - d.x, s[4 * i + 1] - d.y) | (pack_e5m2(s[4 * i + 2] - e.x, s[4 * i + 3] - e.y) << 16);
    }
    uint4* o = reinterpret_cast<uint4*>(eb + ((int64_t)nb * ng + g) * SG_B_GROUP);
    constexpr int PLANE = SG_B_PLANE / 16, HALF = PLANE / 2;            // 16-byte units: plane, K chunk
    const int row_c = (int)(chunk * HALF + kf), row_s = row_c + SG_F;   // rows (k,cos), (k,sin)
    o[row_c] = make_uint4(ch[0], ch[1], ch[2], ch[3]);
    o[row_s] = make_uint4(sh[0], sh[1], sh[2], sh[3]);
    o[PLANE + row_c] = make_uint4(c8h[0], c8h[1], c8l[0], c8l[1]);      // E_8 = [e5m2(E_hi) | e5m2(E_lo)]
    o[PLANE + row_s] = make_uint4(s8h[0], s8h[1], s8l[0], s8l[1]);
}

// CC - n/2 and CS once per frequency (eq. (8); SS = Nt - CC, :130): ws_v[split][4][Nf], planes 2, 3 (0, 1 unused).
// One warp per (frequency, time split): lane = sample mod 32, fp32 partials, fixed shuffle tree (deterministic).
// grid (ceil(Nf / 8), nsplit), 256 threads.
__global__ void __launch_bounds__(256) shared_v_kernel(const ulonglong2* __restrict__ recB, int64_t Nt, int64_t Nf, int64_t split_len, float* __restrict__ ws_v)
{
    pdl_trigger();                                          // (the kernels of a shared-time call are launched as programmatic dependents:
    pdl_wait();                                             //  launch and set-up overlap the predecessor's tail; nothing is read or written before this)
    const int64_t k = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    const unsigned lane = threadIdx.x & 31u;
    const int sp = blockIdx.y;
    if (k >= Nf) return;
    const int64_t j1 = min(Nt, (int64_t)(sp + 1) * split_len);
    float cc = 0.f, cs = 0.f;
    for (int64_t j = (int64_t)sp * split_len + lane; j < j1; j += 32) {
        const ulonglong2 r = __ldg(recB + j);
        const u64 ph = r.x + (u64)k * r.y;                              // u + k v (mod 1, exact 64-bit wrap; reading G3)
        float c, s;
        sincos_phase32((unsigned)((ph + 0x80000000ull) >> 32), c, s);
        cc += fmaf(c, c, -0.5f);
        cs = fmaf(c, s, cs);
    }
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) { cc += __shfl_down_sync(0xffffffffu, cc, o); cs += __shfl_down_sync(0xffffffffu, cs, o); }
    if (lane == 0) {
        ws_v[((int64_t)sp * 4 + 2) * Nf + k] = cc;
        ws_v[((int64_t)sp * 4 + 3) * Nf + k] = cs;
    }
}

// ------------------------------------------------------------------ X tiles
// grid (nmb, ng), 256 threads: row = tid & 127 (series b = 128 nmb + row), chunk = tid >> 7.
__global__ void __launch_bounds__(256) shared_x_kernel(const float* __restrict__ x_in, int64_t x_stride, const double* __restrict__ part_sum,
                                                       const double* __restrict__ part_var, int nparts,
                                                       int64_t B, int64_t Nt, unsigned char* __restrict__ xa, int ng)
{
    pdl_trigger();                                          // (the kernels of a shared-time call are launched as programmatic dependents:
    pdl_wait();                                             //  launch and set-up overlap the predecessor's tail; nothing is read or written before this)
    const int mb = blockIdx.x, g = blockIdx.y;
    const unsigned row = threadIdx.x & 127u, chunk = threadIdx.x >> 7;
    const int64_t b = (int64_t)mb * SG_M + row;
    float x[8];
    const float xs = (b < B) ? x_scale(part_var + b * nparts, nparts, Nt) : 0.f;
    double mean = 0.0;
    if (b < B) { for (int i = 0; i < nparts; ++i) mean += part_sum[b * nparts + i]; mean /= (double)Nt; }   // PAPER.md:41, fixed order
    #pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int64_t j = (int64_t)g * SG_KS + chunk * 8 + i;
        x[i] = (b < B && j < Nt) ? (float)((double)__ldg(x_in + b * x_stride + j) - mean) * xs : 0.f;    // X_j rounded to fp32 once (G4)
    }
    unsigned xh[4], x8h[2], x8l[2];
    #pragma unroll
    for (int i = 0; i < 4; ++i) xh[i] = pack_h2(x[2 * i], x[2 * i + 1]);
    #pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float2 a = unpack_h2(xh[2 * i]), c = unpack_h2(xh[2 * i + 1]);
        x8h[i] = pack_e5m2_h2(xh[2 * i]) | (pack_e5m2_h2(xh[2 * i + 1]) << 16);
        x8l[i] = pack_e5m2(x[4 * i] - a.x, x[4 * i + 1] - a.y) | (pack_e5m2(x[4 * i + 2] - c.x, x[4 * i + 3] - c.y) << 16);
    }
    uint4* o = reinterpret_cast<uint4*>(xa + ((int64_t)mb * ng + g) * SG_A_GROUP);
    constexpr int PLANE = SG_A_PLANE / 16, HALF = PLANE / 2;
    const int r = (int)(chunk * HALF + row);
    o[r] = make_uint4(xh[0], xh[1], xh[2], xh[3]);
    o[PLANE + r] = make_uint4(x8l[0], x8l[1], x8h[0], x8h[1]);         // X_8 = [e5m2(X_lo) | e5m2(X_hi)]
}

// ------------------------------------------------------------------ drain / fused steps 6-7 (shared by both GEMM kernels)
// Called by the four drain warps after the accumulators are complete: q4 = TMEM lane quadrant of the warp.
__device__ __forceinline__ void sg_drain(const SharedGemmParams& p, uint32_t tmem, unsigned q4, unsigned lane, int mb, int nb, int sp)
{
    // ===================== drain: thread = TMEM lane = series; 32 consecutive frequencies per tcgen05.ld =====================
    const int64_t b = (int64_t)mb * SG_M + 32u * q4 + lane;
    if (p.vconst) {
        // ---- fused steps 6-7: P[b][k] from this thread's XC (column kf) and XS (column 128 + kf)
        double inv2var = 0.0;
        if (b < p.B) {
            double qv = 0.0;
            for (int i = 0; i < p.nparts; ++i) qv += p.part_var[b * p.nparts + i];
            double var = qv / (double)(p.Nt - 1);                   // sample variance (reading G1)
            const double xs = (double)(float)(1.0 / sqrt(var));     // X was scaled by the fp32 x_scale(): undo it exactly
            var *= xs * xs;
            inv2var = 0.5 / var;
        }
        const float inv2var_f = (float)inv2var;
        u64 best = 0ull;
        const bool p_vec = p.P && ((p.p_stride & 3) == 0) && ((reinterpret_cast<uintptr_t>(p.P) & 15) == 0);
        #pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
            float vc[32], vs[32];
            tmem_ld32(tmem + ((32u * q4) << 16) + 32u * cc, vc);
            tmem_ld32(tmem + ((32u * q4) << 16) + 128u + 32u * cc, vs);
            const int64_t k0 = (int64_t)(p.nb0 + nb) * SG_F + cc * 32;
            if (b >= p.B) continue;
            float pf[32];
            // branch-free fp32 pass: the 32 loads and combines pipeline.  Frequencies with R > Nt/2 carry cf.x = NaN, come out
            // as NaN and are redone in fp64 below (rare: f -> 0, aliases of regular sampling).
            bool redo = false;
            #pragma unroll
            for (int i = 0; i < 32; ++i) {
                const int64_t k = min(k0 + i, p.Nf - 1);
                const float4 cf = __ldg(p.vconst_f + k);                // same k for the whole warp: one broadcast load
                const float xc2 = vc[i] * vc[i], xs2 = vs[i] * vs[i], S = xc2 + xs2;
                const float D = fmaf(xc2 - xs2, cf.x, 2.f * vc[i] * vs[i] * cf.y);
                pf[i] = fmaf(fmaxf(S + D, 0.f), cf.z, fmaxf(S - D, 0.f) * cf.w) * inv2var_f;
                redo |= (cf.x != cf.x);
            }
            if (redo) {                                                 // warp-uniform (cf depends on k only)
                #pragma unroll
                for (int i = 0; i < 32; ++i) {
                    const int64_t k = min(k0 + i, p.Nf - 1);
                    if (__ldg(&p.vconst_f[k].x) == __ldg(&p.vconst_f[k].x)) continue;
                    const double XC = (double)vc[i], XS = (double)vs[i];
                    const double xc2 = XC * XC, xs2 = XS * XS, S = xc2 + xs2;
                    const double D = (xc2 - xs2) * __ldg(p.vconst + k) + 2.0 * XC * XS * __ldg(p.vconst + p.Nf + k);
                    pf[i] = (float)((fmax(S + D, 0.0) * __ldg(p.vconst + 2 * p.Nf + k) + fmax(S - D, 0.0) * __ldg(p.vconst + 3 * p.Nf + k)) * inv2var);
                    // R > thr Nt: 1/(Nt + R) < 1/((1 + thr) Nt)
                    // ill-conditioned: listed for refine_kernel, which writes P and enters it in the arg-max; here it counts as 0
                    if (p.list.head && k0 + i < p.Nf && __ldg(p.vconst + 2 * p.Nf + k) * ((1.0 + p.refine_thr) * (double)p.Nt) < 1.0 &&
                        refine_push(p.list, b, k)) pf[i] = 0.f;
                }
            }
            #pragma unroll
            for (int i = 0; i < 32; ++i) {
                const int64_t k = k0 + i;
                if (k < p.Nf) {
                    const u64 key = ((u64)__float_as_uint(fmaxf(pf[i], 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k);
                    best = (key > best) ? key : best;
                }
            }
            if (p.P) {
                float* d = p.P + b * p.p_stride + k0;
                if (p_vec && k0 + 32 <= p.Nf) {
                    #pragma unroll
                    for (int i = 0; i < 32; i += 4) *reinterpret_cast<float4*>(d + i) = make_float4(pf[i], pf[i + 1], pf[i + 2], pf[i + 3]);
                } else {
                    #pragma unroll
                    for (int i = 0; i < 32; ++i) if (k0 + i < p.Nf) d[i] = pf[i];
                }
            }
        }
        if (p.peak_idx && b < p.B) {                                // step 7: order-free packed arg-max, lowest k on ties (reading G9)
            atomicMax(p.peak64 + b, best);
            __threadfence();
            const unsigned done = atomicAdd(p.counter + b, 1u);
            if (done == (unsigned)p.nfb_total - 1u) {               // last frequency block of this series (over all bands): publish
                __threadfence();
                const u64 fin = atomicMax(p.peak64 + b, 0ull);
                p.peak_idx[b] = (int32_t)(0xffffffffu - (unsigned)(fin & 0xffffffffull));
                p.peak_val[b] = __uint_as_float((unsigned)(fin >> 32));
            }
        }
    } else {
    float* dst = p.ws_x + ((b * p.nsplit + sp) * 2) * p.x_row;
    #pragma unroll 1
    for (int cc = 0; cc < 8; ++cc) {
        float v[32];
        tmem_ld32(tmem + ((32u * q4) << 16) + 32u * cc, v);
        const int64_t k0 = (int64_t)(p.nb0 + nb) * SG_F + (cc & 3) * 32;
        float* d = dst + (int64_t)(cc >> 2) * p.x_row + k0;
        if (b < p.B) {
            #pragma unroll
            for (int i = 0; i < 32; i += 4)
                if (k0 + i < p.x_row) *reinterpret_cast<float4*>(d + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
        }
    }
    }
}

// ------------------------------------------------------------------ the GEMM
// grid.x = nmb * nfb * nsplit (frequency block fastest, then series block, then split), SG_THREADS threads,
// SG_SMEM bytes of dynamic shared memory.
__global__ void __launch_bounds__(SG_THREADS, 2) shared_gemm_kernel(const SharedGemmParams p)
{
    extern __shared__ __align__(128) unsigned char sg_smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(sg_smem + SG_STAGES * SG_STAGE_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * SG_STAGES + 1);

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    int unit = blockIdx.x;
    const int nb = unit % p.nfb; unit /= p.nfb;
    const int mb = unit % p.nmb;
    const int sp = unit / p.nmb;
    const int nst = p.groups_per_split / SG_KPS;                        // stage-steps of this split
    const int g0 = sp * p.groups_per_split;

    const uint32_t s_stage = smem_u32(sg_smem), s_bar = smem_u32(bars);
    const uint32_t bar_acc = s_bar + 8u * (2 * SG_STAGES);
#define SG_FULL(s) (s_bar + 8u * (unsigned)(s))
#define SG_EMPTY(s) (s_bar + 8u * (unsigned)(SG_STAGES + (s)))

    if (tid == 0) {
        for (int s = 0; s < SG_STAGES; ++s) { mbar_init(SG_FULL(s), 1); mbar_init(SG_EMPTY(s), 1); }
        mbar_init(bar_acc, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"((uint32_t)SG_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);
    pdl_trigger();
    pdl_wait();                                                         // the operand tiles of this band are complete

    if (w == 0) {
        if (lane == 0) {
            // ===================== TMA: the pre-tiled operands, two bulk copies per stage =====================
            const unsigned char* xa = p.xa + ((int64_t)mb * p.ng + g0) * SG_A_GROUP;
            const unsigned char* eb = p.eb + ((int64_t)nb * p.ng + g0) * SG_B_GROUP;
            for (int it = 0; it < nst; ++it) {
                const int s = it & (SG_STAGES - 1);
                const uint32_t ph = (uint32_t)(it / SG_STAGES) & 1u;
                mbar_wait(SG_EMPTY(s), ph ^ 1u);
                const uint32_t st = s_stage + (uint32_t)s * SG_STAGE_BYTES;
                mbar_expect_tx(SG_FULL(s), SG_STAGE_BYTES);
                tma_bulk_g2s(st, xa + (int64_t)it * (SG_KPS * SG_A_GROUP), SG_KPS * SG_A_GROUP, SG_FULL(s));
                tma_bulk_g2s(st + SG_KPS * SG_A_GROUP, eb + (int64_t)it * (SG_KPS * SG_B_GROUP), SG_KPS * SG_B_GROUP, SG_FULL(s));
            }
        }
    } else if (w == 1) {
        if (lane == 0) {
            // ===================== the MMA-issuing thread =====================
            for (int it = 0; it < nst; ++it) {
                const int s = it & (SG_STAGES - 1);
                const uint32_t ph = (uint32_t)(it / SG_STAGES) & 1u;
                mbar_wait(SG_FULL(s), ph);
                tc_fence_after();
                #pragma unroll
                for (int kk = 0; kk < SG_KPS; ++kk) {
                    const uint32_t a0 = s_stage + (uint32_t)s * SG_STAGE_BYTES + kk * SG_A_GROUP;
                    const uint32_t b0 = s_stage + (uint32_t)s * SG_STAGE_BYTES + SG_KPS * SG_A_GROUP + kk * SG_B_GROUP;
                    const uint64_t dAh = umma_desc(a0, SG_A_PLANE / 2, 128), dA8 = umma_desc(a0 + SG_A_PLANE, SG_A_PLANE / 2, 128);
                    const uint64_t dBh = umma_desc(b0, SG_B_PLANE / 2, 128), dB8 = umma_desc(b0 + SG_B_PLANE, SG_B_PLANE / 2, 128);
                    tc_mma_f16(tmem, dAh, dBh, SG_IDESC, (it > 0 || kk > 0) ? 1u : 0u);
                    tc_mma_f8(tmem, dA8, dB8, SG_IDESC | UMMA_IDESC_E5M2, 1u);
                }
                tc_commit(SG_EMPTY(s));
            }
            tc_commit(bar_acc);
        }
    } else {
        // ===================== drain: thread = TMEM lane = series; 32 consecutive frequencies per tcgen05.ld =====================
        mbar_wait(bar_acc, 0u);
        tc_fence_after();
        sg_drain(p, tmem, w & 3u, lane, mb, nb, sp);
        tc_fence_before();
    }
#undef SG_FULL
#undef SG_EMPTY

    __syncwarp();
    tc_fence_before();
    __syncthreads();
    if (w == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((uint32_t)SG_TMEM_COLS) : "memory");
    }
}

}  // namespace lsp
