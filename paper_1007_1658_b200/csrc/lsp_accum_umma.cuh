// lsp_accum_umma.cuh -- steps 3-5 of the hot path on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// Same algebra as lsp_accum_mma.cuh: with k = kb + 128 l + h (h < 128 fine, l < 128 coarse) the phase of
// term (j, k) is a SUM, th_jk = a_jh + b_jl, a_jh = 2 pi frac(u_j + (kb + h) v_j), b_jl = 2 pi frac(128 l v_j)
// (u, v: the exact 64-bit fixed-point turns of lsp_prepass.cuh, reading G3), so the sums of eq. (8)
// are two complex matrix products over the sample index j:
//     W[h,l] = XC + i XS          = sum_j (X_j e^{i a_jh}) (e^{i b_jl})
//     V[h,l] = (CC - SS) + 2i CS  = sum_j (e^{2i a_jh})    (e^{2i b_jl})          (SS = Nt - CC)
// As real GEMMs D[m][n] = sum_k A[m][k] B[n][k]:  rows m = h;  K index = (sample j, component);
//     A_W[h][(j,.)] = (X cos a, X sin a)            A_V[h][(j,.)] = (cos^2 a - 1/2, cos a sin a) = e^{2ia}/2
//     B[(l,Re)][(j,.)] = (cos b, -sin b)            B[(l,Im)][(j,.)] = (sin b, cos b)     (same with 2b for V)
// so D_W[h][(l,Re)] = XC, D_W[h][(l,Im)] = XS, D_V[h][(l,Re)] = CC - n/2, D_V[h][(l,Im)] = CS.
//
// One CTA per SM owns 128 x 128 = 16,384 frequencies over one split of the time axis.  Per k-step of 8
// samples (MMA K = 16 fp16) it issues four tcgen05.mma.cta_group::1.kind::f16 of shape M = 128, N = 256:
//     D_W += A_hi B_hi;  D_W += A_lo B_hi;  D_W += A_hi B_lo;  D_V += A_V B_V
// (fp16 hi + lo pairs carry 22 significant bits; the dropped A_lo B_lo term is 2^-22; V is needed only
// to ~1e-3 of sqrt(Nt) against Nt and takes one pass).  Accumulators: fp32 in TMEM, D_W columns 0..255,
// D_V columns 256..511 -- all 512 columns.  Nothing is loaded by the MMA operands' path from HBM: both
// operand tiles are GENERATED (step 3: integer phase -> MUFU sin/cos) by 16 producer warps
// straight into shared memory in the canonical no-swizzle K-major core-matrix layout, 128 + 128 sincos per
// sample for 16,384 terms.  A ring of NS stages decouples the producers from the single MMA-issuing thread
// (mbarrier full/empty; tcgen05.commit frees a stage).
//
// Step 5 (the chunked sums of PAPER.md:122): tensor-core accumulation rounds toward zero, so D_W is
// drained every `flush_ksteps` k-steps (default 2,048 samples): tcgen05.ld -> fp32 add (round to nearest)
// into the CTA's own slice of `ws` (L2-resident; first drain stores, later ones read-modify-write; no
// atomics, deterministic).  D_V only needs Nt-relative accuracy and is drained once, at the end.
#pragma once
#include "lsp_common.cuh"
#include "lsp_accum.cuh"
#include "lsp_accum_mma.cuh"
#include <cuda_fp16.h>
#include <cuda_fp8.h>

namespace lsp {

constexpr int REC_UMMA = 5;
constexpr int UM_H = 128;                              // fine index h: MMA rows
constexpr int UM_L = 128;                              // coarse index l: MMA columns (l,Re), (l,Im) -> N = 256
constexpr int UM_FPB = UM_H * UM_L;                    // frequencies per CTA
constexpr int UM_KS = 8;                               // samples per k-step
constexpr int UM_TS = 128;                             // samples per record tile (16 k-steps)
constexpr int UM_GEN_WARPS = 16;                       // producer (and drain) warps; warp 16 issues the MMAs
constexpr int UM_THREADS = (UM_GEN_WARPS + 1) * 32;
constexpr int UM_A_BYTES = UM_H * 32;                  // one A operand tile: 128 rows x 16 fp16
constexpr int UM_B_BYTES = 2 * UM_L * 32;              // one B operand tile: 256 rows x 16 fp16
constexpr int UM_STAGE_BYTES = 3 * UM_A_BYTES + 3 * UM_B_BYTES;
constexpr int UM_STAGES = 5;
constexpr int UM_REC_BYTES = 2 * UM_TS * 16;
constexpr size_t UM_SMEM = (size_t)UM_STAGES * UM_STAGE_BYTES + UM_REC_BYTES + 256;
constexpr int UM_TMEM_COLS = 512;

struct UmmaParams {
    const float4* recA;
    const ulonglong2* recB;
    const double* part_var;     // [B][nparts]
    float* ws;                  // [B][nsplit][4][Nf]
    int64_t Nt, Nf;
    int64_t split_len;          // samples per split (multiple of UM_TS)
    int nsplit, nfb, nparts;
    int flush_ksteps;           // k-steps between drains of D_W
    float trunc_ulps;           // pair2 form: expected truncation loss per k-step in ulps of the accumulator, added back at each drain (0: off)
    int unit_x;                 // 1: recA.x is a unit weight, not a measurement: no variance scaling (second pass of the generalised periodogram)
};

// ------------------------------------------------------------------ PTX wrappers (sm_100a)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) { }
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar)          // arrives on `bar` when all earlier MMAs of this thread are done
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]; kind::f16 (fp16 operands, fp32 accumulate); issued by ONE thread.
__device__ __forceinline__ void tc_mma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// Same with kind::f8f6f4 (8-bit float operands, K = 32 per instruction, twice the fp16 rate, fp32 accumulate).
__device__ __forceinline__ void tc_mma_f8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// Shared-memory matrix descriptor, K-major, no swizzle: core matrix = 8 rows x 16 bytes, rows 16 B apart;
// LBO = byte distance between the two 16-byte K chunks, SBO = byte distance between 8-row groups.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}
// Instruction descriptor: D = F32 (bits 4-5 = 1), A = B = F16 (0), both K-major, N >> 3 at bit 17, M >> 4 at bit 24.
constexpr uint32_t UM_IDESC = (1u << 4) | ((uint32_t)(2 * UM_L >> 3) << 17) | ((uint32_t)(UM_H >> 4) << 24);
// kind::f8f6f4: A format at bit 7, B format at bit 10; 1 = E5M2 (the upper byte of an fp16: same exponent range).
constexpr uint32_t UM_IDESC_F8 = UM_IDESC | (1u << 7) | (1u << 10);

// Two fp32 (or one packed fp16 pair) -> two e5m2 bytes in the low 16 bits, round to nearest, first value in the low byte.
__device__ __forceinline__ unsigned pack_e5m2(float a, float b)
{
    return (unsigned)__nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E5M2);
}
__device__ __forceinline__ unsigned pack_e5m2_h2(unsigned h2)
{
    __half2_raw r; r.x = (unsigned short)(h2 & 0xFFFFu); r.y = (unsigned short)(h2 >> 16);
    return (unsigned)__nv_cvt_halfraw2_to_fp8x2(r, __NV_SATFINITE, __NV_E5M2);
}

// 32 lanes x 32 consecutive columns of fp32 accumulators -> 32 registers per thread (lane = TMEM lane).
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32])
{
    uint32_t r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                   "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    #pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void sts128(uint32_t saddr, unsigned a, unsigned b, unsigned c, unsigned d)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" :: "r"(saddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ------------------------------------------------------------------ step 3: operand generation
// One A item: row h, K chunk `c` (4 samples) of the k-step whose records start at rec[s0].  Writes the
// 16-byte row chunks of A_hi, A_lo (X e^{ia} as fp16 hi + lo) and A_V (e^{2ia}/2).
//
// F8 = true (the "8-bit correction" form): the two first-order correction products A_lo B_hi + A_hi B_lo only need
// ~3 significant bits each (they are 2^-12 of the main product), so they are issued as ONE kind::f8f6f4 MMA of
// K = 32: plane 1 then holds, per 16-byte chunk, [e5m2(A_lo) of 4 samples | e5m2(A_hi) of 4 samples] and the matching
// B plane [e5m2(B_hi) | e5m2(B_lo)].  Residual error ~2^-3 * 2^-12 per product, random sign.
template <bool TAIL, bool F8>
__device__ __forceinline__ void um_gen_a(const float4* rec, int s0, unsigned h, uint32_t sA, int nvalid)
{
    unsigned hi[4], lo[4], vv[4], h8[4];
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
        if (F8) { lo[i] = pack_e5m2(lc, ls); h8[i] = pack_e5m2_h2(hi[i]); }
        else lo[i] = pack_h2(lc, ls);
        float v0, v1;
        unpack2(fma2(pack2(c, c), cs, pack2(-0.5f, 0.f)), v0, v1);      // (cos^2 a - 1/2, cos a sin a) = e^{2ia} / 2
        vv[i] = pack_h2(v0, v1);
        if (TAIL && i >= nvalid) vv[i] = 0u;                            // pads (X = 0) must not count in V either
    }
    sts128(sA, hi[0], hi[1], hi[2], hi[3]);
    if (F8) sts128(sA + UM_A_BYTES, lo[0] | (lo[1] << 16), lo[2] | (lo[3] << 16), h8[0] | (h8[1] << 16), h8[2] | (h8[3] << 16));
    else sts128(sA + UM_A_BYTES, lo[0], lo[1], lo[2], lo[3]);
    sts128(sA + 2 * UM_A_BYTES, vv[0], vv[1], vv[2], vv[3]);
}
template <bool F8 = false>
__device__ __forceinline__ void um_gen_a(const float4* rec, int s0, unsigned h, uint32_t sA, int64_t left)
{
    if (left >= 4) um_gen_a<false, F8>(rec, s0, h, sA, 4);              // `left` is warp-uniform
    else um_gen_a<true, F8>(rec, s0, h, sA, (int)max((int64_t)0, left));
}

// One B item: coarse index l, K chunk `c`: rows (l,Re) and (l,Im) of B_hi, B_lo (e^{ib}) and B_V (e^{2ib}).
__device__ __forceinline__ void um_gen_b(const float4* rec, int s0, unsigned l, uint32_t sB)
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
    sts128(sB, rh[0], rh[1], rh[2], rh[3]);
    sts128(sB + UM_L * 16, ih[0], ih[1], ih[2], ih[3]);
    sts128(sB + UM_B_BYTES, rl[0], rl[1], rl[2], rl[3]);
    sts128(sB + UM_B_BYTES + UM_L * 16, il[0], il[1], il[2], il[3]);
    sts128(sB + 2 * UM_B_BYTES, rv[0], rv[1], rv[2], rv[3]);
    sts128(sB + 2 * UM_B_BYTES + UM_L * 16, iv[0], iv[1], iv[2], iv[3]);
}

// ------------------------------------------------------------------ step 5: drain 64 accumulator columns into ws
// Thread = TMEM lane = row h; its 64 registers are 64 consecutive coarse indices l.  For a fixed column the 32
// lanes of the warp touch 32 consecutive frequencies (k = kb + 128 l + h): coalesced 128-byte accesses.
__device__ __forceinline__ void um_drain64(uint32_t taddr, float* dst, int64_t k0, int64_t Nf, bool first)
{
    #pragma unroll 1
    for (int half = 0; half < 2; ++half) {
        float v[32];
        tmem_ld32(taddr + 32u * half, v);
        const int64_t kh = k0 + (int64_t)half * 32 * UM_H;
        if (!first) {
            #pragma unroll
            for (int i = 0; i < 32; ++i) { const int64_t k = kh + (int64_t)i * UM_H; if (k < Nf) v[i] += dst[k]; }
        }
        #pragma unroll
        for (int i = 0; i < 32; ++i) { const int64_t k = kh + (int64_t)i * UM_H; if (k < Nf) dst[k] = v[i]; }
    }
}

// ------------------------------------------------------------------ the kernel
// grid.x = B * nsplit * nfb (frequency block fastest), UM_THREADS threads, UM_SMEM bytes of dynamic shared memory,
// one CTA per SM (it owns all 512 TMEM columns).
__global__ void __launch_bounds__(UM_THREADS, 1) accum_umma_kernel(const UmmaParams p)
{
    extern __shared__ __align__(128) unsigned char um_smem[];
    float4* rec = reinterpret_cast<float4*>(um_smem + UM_STAGES * UM_STAGE_BYTES);                 // [2][UM_TS] {X/sigma, pA32, v32, w32}
    uint64_t* bars = reinterpret_cast<uint64_t*>(um_smem + UM_STAGES * UM_STAGE_BYTES + UM_REC_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * UM_STAGES + 2);

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t b = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * UM_FPB;
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const int64_t n_samp = j_end - j_begin;
    const int nks = (int)((n_samp + UM_KS - 1) / UM_KS);
    const int flush_ksteps = max(1, p.flush_ksteps);

    const uint32_t s_stage = smem_u32(um_smem), s_bar = smem_u32(bars);
    const uint32_t bar_accf = s_bar + 8u * (2 * UM_STAGES), bar_acce = bar_accf + 8u;
#define UM_FULL(s) (s_bar + 8u * (unsigned)(s))
#define UM_EMPTY(s) (s_bar + 8u * (unsigned)(UM_STAGES + (s)))

    if (tid == 0) {
        for (int s = 0; s < UM_STAGES; ++s) { mbar_init(UM_FULL(s), UM_GEN_WARPS); mbar_init(UM_EMPTY(s), 1); }
        mbar_init(bar_accf, 1);
        mbar_init(bar_acce, UM_GEN_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == UM_GEN_WARPS) {                                            // the MMA warp owns the TMEM allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"((uint32_t)UM_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);

    if (w < UM_GEN_WARPS) {
        // ===================== producers: steps 3 (operand tiles) and 5 (drain) =====================
        const float4* recA = p.recA + b * p.Nt;
        const ulonglong2* recB = p.recB + b * p.Nt;
        const float xs = (tid < UM_TS) ? (p.unit_x ? 1.f : x_scale(p.part_var + b * p.nparts, p.nparts, p.Nt)) : 0.f;
        float pre_x = 0.f; u64 pre_u = 0ull, pre_v = 0ull; bool pre_ok = false;
        auto prefetch = [&](int ti) {
            const int64_t j = j_begin + (int64_t)ti * UM_TS + tid;
            pre_ok = (tid < UM_TS) && (j < j_end);
            if (pre_ok) { pre_x = __ldg(&recA[j].x); const ulonglong2 q = __ldg(recB + j); pre_u = q.x; pre_v = q.y; }
        };
        prefetch(0);
        const bool is_b = w < UM_GEN_WARPS / 2;                         // warps 0-7: B items, 8-15: A items
        const unsigned idx = tid & 127u;                                // l (B) or h (A)
        const int chunk = (int)((tid >> 7) & 1u);                       // which 4 samples of the k-step
        const unsigned q4 = w & 3u, cg = w >> 2;                        // drain: TMEM lane quadrant, column group
        float* ws_unit = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
        const int64_t k0 = kb + (int64_t)(64u * (cg & 1u)) * UM_H + (int64_t)(32u * q4 + lane);
        const uint32_t t_drain = tmem + ((32u * q4) << 16) + 64u * cg;
        int kin = 0, flushes = 0;

        for (int ks = 0; ks < nks; ++ks) {
            const int s = ks % UM_STAGES;
            const uint32_t ph = (uint32_t)(ks / UM_STAGES) & 1u;
            const int ti = ks >> 4;
            if ((ks & 15) == 0) {                                       // next record tile (buffer ti & 1)
                if (tid < UM_TS) {
                    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);         // pad: X = 0, phases 0
                    if (pre_ok) {
                        const u64 pa = pre_u + (u64)kb * pre_v;         // u + kb v (mod 1, 64-bit wrap; reading G3)
                        r.x = pre_x * xs;
                        r.y = __uint_as_float((unsigned)((pa + 0x80000000ull) >> 32));
                        r.z = __uint_as_float((unsigned)((pre_v + 0x80000000ull) >> 32));
                        r.w = __uint_as_float((unsigned)(((u64)UM_H * pre_v + 0x80000000ull) >> 32));
                    }
                    rec[(ti & 1) * UM_TS + tid] = r;
                    prefetch(ti + 1);
                }
                asm volatile("bar.sync 1, %0;" :: "n"(UM_GEN_WARPS * 32) : "memory");
            }
            mbar_wait(UM_EMPTY(s), ph ^ 1u);                            // the MMAs that read this stage have completed
            const float4* rt = rec + (ti & 1) * UM_TS;
            const int s0 = (ks & 15) * UM_KS + chunk * 4;
            const uint32_t st = s_stage + (uint32_t)s * UM_STAGE_BYTES;
            if (is_b) {
                um_gen_b(rt, s0, idx, st + 3 * UM_A_BYTES + chunk * (UM_B_BYTES / 2) + idx * 16);
            } else {
                um_gen_a(rt, s0, idx, st + chunk * (UM_A_BYTES / 2) + idx * 16, n_samp - ((int64_t)ks * UM_KS + chunk * 4));
            }
            fence_proxy_async();                                        // generic-proxy stores -> visible to the tensor core
            __syncwarp();
            if (lane == 0) mbar_arrive(UM_FULL(s));

            const bool last = (ks == nks - 1);
            if (++kin == flush_ksteps || last) {
                mbar_wait(bar_accf, (uint32_t)flushes & 1u);            // every MMA issued so far has completed
                tc_fence_after();
                um_drain64(t_drain, ws_unit + (int64_t)(cg >> 1) * p.Nf, k0, p.Nf, flushes == 0);
                if (last) um_drain64(t_drain + 256u, ws_unit + (int64_t)(2 + (cg >> 1)) * p.Nf, k0, p.Nf, true);
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
            const int s = ks % UM_STAGES;
            const uint32_t ph = (uint32_t)(ks / UM_STAGES) & 1u;
            mbar_wait(UM_FULL(s), ph);
            tc_fence_after();
            const uint32_t a0 = s_stage + (uint32_t)s * UM_STAGE_BYTES, b0 = a0 + 3 * UM_A_BYTES;
            const uint64_t dAh = umma_desc(a0, UM_A_BYTES / 2, 128), dAl = umma_desc(a0 + UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dAv = umma_desc(a0 + 2 * UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dBh = umma_desc(b0, UM_B_BYTES / 2, 128), dBl = umma_desc(b0 + UM_B_BYTES, UM_B_BYTES / 2, 128);
            const uint64_t dBv = umma_desc(b0 + 2 * UM_B_BYTES, UM_B_BYTES / 2, 128);
            tc_mma_f16(tmem, dAh, dBh, UM_IDESC, kin > 0 ? 1u : 0u);
            tc_mma_f16(tmem, dAl, dBh, UM_IDESC, 1u);
            tc_mma_f16(tmem, dAh, dBl, UM_IDESC, 1u);
            tc_mma_f16(tmem + 256u, dAv, dBv, UM_IDESC, ks > 0 ? 1u : 0u);
            tc_commit(UM_EMPTY(s));
            const bool last = (ks == nks - 1);
            if (++kin == flush_ksteps || last) {
                tc_commit(bar_accf);
                if (!last) { mbar_wait(bar_acce, (uint32_t)flushes & 1u); tc_fence_after(); }
                ++flushes; kin = 0;
            }
        }
    }
#undef UM_FULL
#undef UM_EMPTY

    tc_fence_before();
    __syncthreads();
    if (w == UM_GEN_WARPS) {
        __syncwarp();
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((uint32_t)UM_TMEM_COLS) : "memory");
    }
}

}  // namespace lsp
