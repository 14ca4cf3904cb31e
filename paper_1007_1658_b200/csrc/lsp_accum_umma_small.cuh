// lsp_accum_umma_small.cuh -- the tcgen05 form of steps 3-5 for SHORT frequency grids (lsp_tc.cuh states the algebra).
//
// A CTA owns 128 fine x L coarse frequencies, k = kb + 128 l + h, with the coarse extent L a template parameter
// (16, 32 or 64): the MMAs are m128 n(2L) k16 and the accumulators take 4L of the 512 TMEM columns (D_W: columns
// [0, 2L), D_V: [2L, 4L)), so two (L = 16: three) CTAs of 8 producer warps + 1 MMA warp share an SM: one CTA's set-up
// and drain overlap the others' main loops, and the extra warps hide the latency of the generation chain
// (LDS -> IMAD -> I2F -> MUFU -> F2FP -> STS).  As real GEMMs D[m][n] = sum_k A[m][k] B[n][k], K index = (sample j, component):
//     A_W[h][(j,.)] = (X cos a, X sin a)            A_V[h][(j,.)] = (cos^2 a - 1/2, cos a sin a) = e^{2ia}/2
//     B[(l,Re)][(j,.)] = (cos b, -sin b)            B[(l,Im)][(j,.)] = (sin b, cos b)     (same with 2b for V)
// so D_W[h][(l,Re)] = XC, D_W[h][(l,Im)] = XS, D_V[h][(l,Re)] = CC - n/2, D_V[h][(l,Im)] = CS.  Per k-step of 8 samples:
//     D_W += A_hi B_hi;  D_W += A_lo B_hi;  D_W += A_hi B_lo;  D_V += A_V B_V          (four kind::f16 MMAs)
// Both operand tiles are GENERATED (step 3: integer phase -> MUFU sin/cos) by the producer warps straight
// into shared memory in the canonical no-swizzle K-major core-matrix layout; the coarse operand B (2L rows) by a
// rotating subset of the producer threads.  A ring of stages decouples the producers from the single MMA-issuing thread
// (mbarrier full/empty; tcgen05.commit frees a stage).  With L <= 32 the kernel is bound by the generation of the
// fine operand A (128 MUFU sin/cos pairs per sample for 128 L terms), not by the tensor pipe.
//
// Step 5 (the chunked sums of PAPER.md:122): tensor-core accumulation rounds toward zero, so D_W is drained every
// `flush_ksteps` k-steps (default 2,048 samples): tcgen05.ld -> the expected truncation loss of the window added back
// (tc_trunc_comp, lsp_tc.cuh) -> fp32 add (round to nearest) into the CTA's own slice of
// `ws` (L2-resident; first drain stores, later ones read-modify-write; no atomics, deterministic).  D_V only needs
// Nt-relative accuracy and is drained once, at the end.
#pragma once
#include "lsp_tc.cuh"

namespace lsp {

// One A item: row h, 4 samples starting at rec[s0].  Writes the 16-byte row chunks of A_hi, A_lo (X e^{ia} as
// fp16 hi + lo) and A_V (e^{2ia}/2).
template <bool TAIL, bool WEIGHTED = false>
__device__ __forceinline__ void um_gen_a(const float4* rec, int s0, unsigned h, uint32_t sA, int nvalid, const float* recw = nullptr)
{
    unsigned hi[4], lo[4], vv[4];
    #pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float4 r = rec[s0 + i];                                   // {X / sigma, pA32, v32, w32}: broadcast read
        float c, s;
        sincos_phase32(__float_as_uint(r.y) + h * __float_as_uint(r.z), c, s);
        const u64 cs = pack2(c, s);
        float xc, xs;
        unpack2(mul2(pack2(r.x, r.x), cs), xc, xs);                     // packed FP32: one FMUL2
        hi[i] = pack_h2(xc, xs);
        const float2 hf = unpack_h2(hi[i]);
        float lc, ls;
        unpack2(fma2(pack2(hf.x, hf.y), pack2(-1.f, -1.f), pack2(xc, xs)), lc, ls);
        lo[i] = pack_h2(lc, ls);
        float v0, v1;
        unpack2(fma2(pack2(c, c), cs, pack2(-0.5f, 0.f)), v0, v1);      // (cos^2 a - 1/2, cos a sin a) = e^{2ia} / 2
        if (WEIGHTED) { const float wv = recw[s0 + i]; v0 *= wv; v1 *= wv; }   // V = sum_j w_j e^{2i theta} (broadcast read)
        // stochastic rounding; the random bits are the low mantissa bits of X cos a (X is data: they are noise)
        vv[i] = pack_h2_sr(v0, v1, __float_as_uint(xc) & 0x1fffu);
        if (TAIL && i >= nvalid) vv[i] = 0u;                            // pads (X = 0) must not count in V either
    }
    sts128(sA, hi[0], hi[1], hi[2], hi[3]);
    sts128(sA + UM_A_BYTES, lo[0], lo[1], lo[2], lo[3]);
    sts128(sA + 2 * UM_A_BYTES, vv[0], vv[1], vv[2], vv[3]);
}
template <bool WEIGHTED = false>
__device__ __forceinline__ void um_gen_a(const float4* rec, int s0, unsigned h, uint32_t sA, int64_t left, const float* recw = nullptr)
{
    if (left >= 4) um_gen_a<false, WEIGHTED>(rec, s0, h, sA, 4, recw);                  // `left` is warp-uniform
    else um_gen_a<true, WEIGHTED>(rec, s0, h, sA, (int)max((int64_t)0, left), recw);
}

constexpr int US_GEN_WARPS = 8;                        // producer (and drain) warps; warp 8 issues the MMAs
constexpr int US_THREADS = (US_GEN_WARPS + 1) * 32;

template <int L, int US_STAGES> struct UmmaSmall {
    static constexpr int B_BYTES = 2 * L * 32;         // one B operand tile: 2L rows x 16 fp16
    static constexpr int STAGE_BYTES = 3 * UM_A_BYTES + 3 * B_BYTES;
    static constexpr size_t SMEM = (size_t)US_STAGES * STAGE_BYTES + UM_REC_BYTES + UM_RECW_BYTES + 256;
    static constexpr int TMEM_COLS = 4 * L < 32 ? 32 : 4 * L;
    static constexpr uint32_t IDESC = umma_idesc(UM_H, 2 * L);
    static constexpr int FPB = UM_H * L;               // frequencies per CTA
};

// One B item: coarse index l, K chunk of 4 samples: rows (l,Re) and (l,Im) of B_hi, B_lo (e^{ib}) and B_V (e^{2ib}).
template <int L>
__device__ __forceinline__ void us_gen_b(const float4* rec, int s0, unsigned l, uint32_t sB)
{
    unsigned rh[4], ih[4], rl[4], il[4], rv[4], iv[4];
    #pragma unroll
    for (int i = 0; i < 4; ++i) {
        float c, s;
        sincos_phase32(l * __float_as_uint(rec[s0 + i].w), c, s);
        rh[i] = pack_h2(c, -s);
        ih[i] = pack_h2(s, c);
        const float2 hf = unpack_h2(rh[i]);                             // (c_h, -s_h)
        const float dc = c - hf.x, ds = s + hf.y;
        rl[i] = pack_h2(dc, -ds);
        il[i] = pack_h2(ds, dc);
        const float cc = c + c, c2 = fmaf(cc, c, -1.f), s2 = cc * s;
        rv[i] = pack_h2(c2, -s2);
        iv[i] = pack_h2(s2, c2);
    }
    constexpr int BB = 2 * L * 32;                                      // bytes of one B operand tile
    sts128(sB, rh[0], rh[1], rh[2], rh[3]);
    sts128(sB + L * 16, ih[0], ih[1], ih[2], ih[3]);
    sts128(sB + BB, rl[0], rl[1], rl[2], rl[3]);
    sts128(sB + BB + L * 16, il[0], il[1], il[2], il[3]);
    sts128(sB + 2 * BB, rv[0], rv[1], rv[2], rv[3]);
    sts128(sB + 2 * BB + L * 16, iv[0], iv[1], iv[2], iv[3]);
}

// Drain L accumulator columns (one of Re / Im) of this warp's 32 TMEM lanes into one plane of ws.
// Thread = TMEM lane = row h; column l is frequency k0 + 128 l: for a fixed column the warp touches
// 32 consecutive frequencies (coalesced).
// n_ksteps > 0: D_W of a drain window of that many k-steps: the expected truncation loss is added back (tc_trunc_comp; three fp16 MMAs
// per k-step add into D_W here); 0: no compensation (D_V).
template <int L>
__device__ __forceinline__ void us_drain(uint32_t taddr, float* dst, int64_t k0, int64_t Nf, bool first, float n_ksteps = 0.f, float inv_coherent = 0.f)
{
    #pragma unroll 1
    for (int part = 0; part < L / 16; ++part) {
        float v[16];
        tmem_ld16(taddr + 16u * part, v);
        if (n_ksteps > 0.f) {
            #pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = tc_trunc_comp(v[i], n_ksteps, 1.125f, inv_coherent);
        }
        const int64_t kp = k0 + (int64_t)part * 16 * UM_H;
        if (!first) {
            #pragma unroll
            for (int i = 0; i < 16; ++i) { const int64_t k = kp + (int64_t)i * UM_H; if (k < Nf) v[i] += dst[k]; }
        }
        #pragma unroll
        for (int i = 0; i < 16; ++i) { const int64_t k = kp + (int64_t)i * UM_H; if (k < Nf) dst[k] = v[i]; }
    }
}

// grid.x = B * nsplit * nfb (frequency block fastest), US_THREADS threads, UmmaSmall<L, US_STAGES>::SMEM bytes of
// dynamic shared memory (one k-step of 8 samples per stage), MINB CTAs per SM.  p.nfb = ceil(Nf / (128 L)).
// FUSED_PRE (one launch fewer where launches are what a call costs: C1, C2): steps 1-2 run inside this kernel.  Every CTA forms
// the mean and the variance of its (short) series itself -- the same fixed-order fp64 reduction in every CTA, so all of them, and
// the finish step through part_var_out, use bit-identical values -- and computes the exact 64-bit phases (reading G3) of the
// samples of its own time split while it stages them.  The tensor forms need no per-sample rotation (cos d, sin d), so the fp64
// work per sample is two exact products.
// WEIGHTED (weighted generalised periodogram, never with FUSED_PRE): X = recA.x recW.x = w_j (x_j - xbar_w) / sigma (w_j in the unit
// pass), and the double-angle operand is scaled by w_j.
template <int L, int US_STAGES, int MINB, bool FUSED_PRE = false, bool WEIGHTED = false>
__global__ void __launch_bounds__(US_THREADS, MINB) accum_umma_small_kernel(const UmmaParams p)
{
    using C = UmmaSmall<L, US_STAGES>;
    extern __shared__ __align__(128) unsigned char um_smem[];
    float4* rec = reinterpret_cast<float4*>(um_smem + US_STAGES * C::STAGE_BYTES);                 // [2][UM_TS] {X/sigma, pA32, v32, w32}
    float* recw = reinterpret_cast<float*>(um_smem + US_STAGES * C::STAGE_BYTES + UM_REC_BYTES);    // [2][UM_TS] normalised weight (WEIGHTED)
    uint64_t* bars = reinterpret_cast<uint64_t*>(um_smem + US_STAGES * C::STAGE_BYTES + UM_REC_BYTES + UM_RECW_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * US_STAGES + 2);

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t b = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * C::FPB;
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const int64_t n_samp = j_end - j_begin;
    const int nks = (int)((n_samp + UM_KS - 1) / UM_KS);
    const int flush_ksteps = max(1, p.flush_ksteps);

    const uint32_t s_stage = smem_u32(um_smem), s_bar = smem_u32(bars);
    const uint32_t bar_accf = s_bar + 8u * (2 * US_STAGES), bar_acce = bar_accf + 8u;
#define US_FULL(s) (s_bar + 8u * (unsigned)(s))
#define US_EMPTY(s) (s_bar + 8u * (unsigned)(US_STAGES + (s)))

    if (tid == 0) {
        for (int s = 0; s < US_STAGES; ++s) { mbar_init(US_FULL(s), US_GEN_WARPS); mbar_init(US_EMPTY(s), 1); }
        mbar_init(bar_accf, 1);
        mbar_init(bar_acce, US_GEN_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == US_GEN_WARPS) {                                            // the MMA warp owns the TMEM allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"((uint32_t)C::TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);

    pdl_trigger();                                                      // the finish kernel may be scheduled (it waits for this grid to complete)
    pdl_wait();                                                         // the pre-pass has completed: records and variance partials are visible
    if (w < US_GEN_WARPS) {
        // ===================== producers: steps 3 (operand tiles) and 5 (drain) =====================
        const float4* recA = p.recA + b * p.Nt;
        const ulonglong2* recB = p.recB + b * p.Nt;
        float xs;
        double mean = 0.0, t0 = 0.0;
        const double* tb = nullptr; const float* xb = nullptr;
        if (FUSED_PRE) {
            // steps 1-2: mean, then sum (x - mean)^2, over the whole series by the 256 producer threads
            tb = p.t + b * p.t_stride; xb = p.x + b * p.x_stride;
            double* red = reinterpret_cast<double*>(rec);               // 8 doubles of scratch (the record tile is not in use yet)
            double a0 = 0.0;
            for (int64_t j = tid; j < p.Nt; j += US_GEN_WARPS * 32) a0 += (double)__ldg(xb + j);
            #pragma unroll
            for (int o = 16; o > 0; o >>= 1) a0 += __shfl_down_sync(0xffffffffu, a0, o);
            if (lane == 0) red[w] = a0;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            double sum = 0.0;
            #pragma unroll
            for (int i = 0; i < US_GEN_WARPS; ++i) sum += red[i];       // fixed order: the same value in every thread of every CTA
            mean = sum / (double)p.Nt;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            double a1 = 0.0;
            for (int64_t j = tid; j < p.Nt; j += US_GEN_WARPS * 32) { const double d = (double)__ldg(xb + j) - mean; a1 += d * d; }
            #pragma unroll
            for (int o = 16; o > 0; o >>= 1) a1 += __shfl_down_sync(0xffffffffu, a1, o);
            if (lane == 0) red[w] = a1;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            double q2 = 0.0;
            #pragma unroll
            for (int i = 0; i < US_GEN_WARPS; ++i) q2 += red[i];
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");   // `red` is the record tile from here on
            if (tid == 0 && sp == 0 && fb == 0) { p.part_var_out[b] = q2; p.part_sum_out[b] = sum; p.peak64[b] = 0ull; p.counter[b] = 0u; }
            xs = (tid < UM_TS) ? x_scale(&q2, 1, p.Nt) : 0.f;           // the finish step recomputes exactly this from part_var_out
            t0 = __ldg(tb);                                             // time origin (reading G6)
        } else {
            xs = (tid < UM_TS) ? (p.unit_x ? 1.f : x_scale(p.part_var + b * p.nparts, p.nparts, p.Nt)) : 0.f;
        }
        float pre_x = 0.f, pre_w = 1.f; u64 pre_u = 0ull, pre_v = 0ull; bool pre_ok = false;
        const float4* recW = WEIGHTED ? p.recW + b * p.Nt : nullptr;
        auto prefetch = [&](int ti) {
            const int64_t j = j_begin + (int64_t)ti * UM_TS + tid;
            pre_ok = (tid < UM_TS) && (j < j_end);
            if (!pre_ok) return;
            if (FUSED_PRE) {
                pre_x = (float)((double)__ldg(xb + j) - mean);          // X_j rounded to fp32 once (G4)
                const double tp = __ldg(tb + j) - t0;
                pre_u = frac_fixed64(p.f_min, tp, nullptr);
                pre_v = frac_fixed64(p.df, tp, nullptr);
            } else { pre_x = __ldg(&recA[j].x); const ulonglong2 q = __ldg(recB + j); pre_u = q.x; pre_v = q.y; }
            if (WEIGHTED) pre_w = __ldg(&recW[j].x);
        };
        prefetch(0);
        const unsigned h = tid & 127u;                                  // A item: row h, 4 samples `chunk` of the k-step
        const int chunk = (int)(tid >> 7);
        const unsigned q4 = w & 3u, part = w >> 2;                      // drain: TMEM lane quadrant, Re (0) / Im (1) columns
        float* ws_unit = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
        const int64_t k0 = kb + (int64_t)(32u * q4 + lane);
        const uint32_t t_drain = tmem + ((32u * q4) << 16) + (uint32_t)L * part;
        int kin = 0, flushes = 0;

        for (int ks = 0; ks < nks; ++ks) {
            const int s = ks % US_STAGES;
            const uint32_t ph = (uint32_t)(ks / US_STAGES) & 1u;
            const int ti = ks >> 4;
            if ((ks & 15) == 0) {                                       // next record tile (buffer ti & 1)
                if (tid < UM_TS) {
                    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);         // pad: X = 0, phases 0
                    if (pre_ok) {
                        const u64 pa = pre_u + (u64)kb * pre_v;         // u + kb v (mod 1, 64-bit wrap; reading G3)
                        r.x = WEIGHTED ? pre_x * xs * pre_w : pre_x * xs;
                        r.y = __uint_as_float((unsigned)((pa + 0x80000000ull) >> 32));
                        r.z = __uint_as_float((unsigned)((pre_v + 0x80000000ull) >> 32));
                        r.w = __uint_as_float((unsigned)(((u64)UM_H * pre_v + 0x80000000ull) >> 32));
                    }
                    rec[(ti & 1) * UM_TS + tid] = r;
                    if (WEIGHTED) recw[(ti & 1) * UM_TS + tid] = pre_ok ? pre_w * pre_w : 0.f;
                    prefetch(ti + 1);
                }
                asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            }
            mbar_wait(US_EMPTY(s), ph ^ 1u);                            // the MMAs that read this stage have completed
            const float4* rt = rec + (ti & 1) * UM_TS;
            const int sb = (ks & 15) * UM_KS;
            const uint32_t st = s_stage + (uint32_t)s * C::STAGE_BYTES;
            um_gen_a<WEIGHTED>(rt, sb + chunk * 4, h, st + chunk * (UM_A_BYTES / 2) + h * 16, n_samp - ((int64_t)ks * UM_KS + chunk * 4), recw + (ti & 1) * UM_TS);
            const unsigned bt = (tid - (unsigned)ks * (2u * L)) & 255u;  // the 2L B items rotate over the 256 producer threads
            if (bt < 2u * L) {
                const unsigned l = bt % (unsigned)L, bc = bt / (unsigned)L;
                us_gen_b<L>(rt, sb + (int)bc * 4, l, st + 3 * UM_A_BYTES + bc * (C::B_BYTES / 2) + l * 16);
            }
            fence_proxy_async();                                        // generic-proxy stores -> visible to the tensor core
            __syncwarp();
            if (lane == 0) mbar_arrive(US_FULL(s));

            const bool last = (ks == nks - 1);
            if (++kin == flush_ksteps || last) {
                mbar_wait(bar_accf, (uint32_t)flushes & 1u);            // every MMA issued so far has completed
                tc_fence_after();
                {
                    const float nk = (float)kin;                        // k-steps of this window
                    us_drain<L>(t_drain, ws_unit + (int64_t)part * p.Nf, k0, p.Nf, flushes == 0, p.trunc_ulps < 0.f ? nk : 0.f,
                                0.6366198f / (16.f * nk * (p.unit_x ? TC_MEAN_ABS_COS : TC_MEAN_ABS_PRODUCT)));
                }
                // D_V is drained with D_W: left to accumulate over the whole split it loses ~n ulp toward zero where sum e^{2i theta} is coherent
                us_drain<L>(t_drain + 2u * L, ws_unit + (int64_t)(2 + part) * p.Nf, k0, p.Nf, flushes == 0);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_acce);
                ++flushes; kin = 0;
            }
        }
    } else if (lane == 0) {
        // ===================== step 4: the single MMA-issuing thread =====================
        int kin = 0, flushes = 0;
        for (int ks = 0; ks < nks; ++ks) {
            const int s = ks % US_STAGES;
            const uint32_t ph = (uint32_t)(ks / US_STAGES) & 1u;
            mbar_wait(US_FULL(s), ph);
            tc_fence_after();
            const uint32_t a0 = s_stage + (uint32_t)s * C::STAGE_BYTES, b0 = a0 + 3 * UM_A_BYTES;
            const uint64_t dAh = umma_desc(a0, UM_A_BYTES / 2, 128), dAl = umma_desc(a0 + UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dAv = umma_desc(a0 + 2 * UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dBh = umma_desc(b0, C::B_BYTES / 2, 128), dBl = umma_desc(b0 + C::B_BYTES, C::B_BYTES / 2, 128);
            const uint64_t dBv = umma_desc(b0 + 2 * C::B_BYTES, C::B_BYTES / 2, 128);
            tc_mma_f16(tmem, dAh, dBh, C::IDESC, kin > 0 ? 1u : 0u);
            tc_mma_f16(tmem, dAl, dBh, C::IDESC, 1u);
            tc_mma_f16(tmem, dAh, dBl, C::IDESC, 1u);
            tc_mma_f16(tmem + 2u * L, dAv, dBv, C::IDESC, kin > 0 ? 1u : 0u);
            tc_commit(US_EMPTY(s));
            const bool last = (ks == nks - 1);
            if (++kin == flush_ksteps || last) {
                tc_commit(bar_accf);
                if (!last) { mbar_wait(bar_acce, (uint32_t)flushes & 1u); tc_fence_after(); }
                ++flushes; kin = 0;
            }
        }
    }
#undef US_FULL
#undef US_EMPTY

    tc_fence_before();
    __syncthreads();
    if (w == US_GEN_WARPS) {
        __syncwarp();
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((uint32_t)C::TMEM_COLS) : "memory");
    }
}

}  // namespace lsp
