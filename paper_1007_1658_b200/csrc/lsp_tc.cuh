// lsp_tc.cuh -- what the tensor-core forms of steps 3-5 share: the factorisation they rest on, operand formats,
// and thin PTX wrappers for sm_100a (mbarrier, cp.async.bulk, tcgen05.mma / commit / ld, cluster scope).
//
// The algebra.  On a uniform grid the phase of term (j, k) is a SUM: with k = kb + H l + h
// (h < H fine, l coarse)   th_jk = a_jh + b_jl,  a_jh = 2 pi frac(u_j + (kb + h) v_j),  b_jl = 2 pi frac(H l v_j)
// (u, v: the exact 64-bit fixed-point turns of lsp_prepass.cuh, reading G3), so the sums of eq. (8)
// are two complex matrix products over the sample index j:
//     W[h,l] = XC + i XS          = sum_j (X_j e^{i a_jh}) (e^{i b_jl})
//     V[h,l] = (CC - SS) + 2i CS  = sum_j (e^{2i a_jh})    (e^{2i b_jl})          (SS = Nt - CC)
// i.e. real GEMMs D[m][n] = sum_k A[m][k] B[n][k] with K index (sample j, component).  H + L sin/cos pairs per sample
// generate H L terms: the angle-addition recurrence of north_star (2), re-anchored from exact integer phases, carried
// out by the tensor pipe.  Every operand element is produced by steps 2-3 (integer phase -> MUFU sin/cos).
//
// Operand precision: fp16 hi + lo (22 significant bits).  D_W += A_hi B_hi (kind::f16) + [A_lo B_hi + A_hi B_lo]; the
// bracket is 2^-12 of the main product and needs ~3 significant bits, so it is either two more fp16 MMAs or ONE
// kind::f8f6f4 MMA of K = 32 on e5m2 operands (the upper byte of an fp16: same exponent range, no scaling).  V needs
// only Nt-relative accuracy: one fp16 MMA.  Accumulators: fp32 in TMEM; the tensor core adds with round-toward-zero, so
// D_W is drained every <= 2,048 samples (8,192 in the CTA-pair form) and the expected loss of the window is added back at the
// drain (tc_trunc_comp below; the paper's chunked sums).
#pragma once
#include "lsp_common.cuh"
#include <cuda_fp16.h>
#include <cuda_fp8.h>

namespace lsp {

constexpr int UM_H = 128;                              // MMA rows per CTA
constexpr int UM_KS = 8;                               // samples per k-step (MMA K = 16 fp16: 8 samples x 2 components)
constexpr int UM_TS = 128;                             // samples per record tile (16 k-steps)
constexpr int UM_A_BYTES = UM_H * 32;                  // one 128-row operand plane of a k-step: 128 rows x 16 fp16
constexpr int UM_REC_BYTES = 2 * UM_TS * 16;           // double-buffered record tile
constexpr int UM_RECW_BYTES = 2 * UM_TS * 4;           // ... and the normalised weights of its samples (weighted generalised periodogram)
constexpr int UM_TMEM_COLS = 512;

struct UmmaParams {
    const float4* recA;
    const ulonglong2* recB;
    const float4* recW;         // weighted generalised periodogram (short-grid and batch kernels): recW[j].x = sqrt of the normalised weight w_j;
                                // recA.x carries one factor sqrt(w_j) already (lsp_prepass.cuh): X = recA.x recW.x, V = sum w e^{2i theta}; else NULL
    const double* part_var;     // [B][nparts]
    float* ws;                  // [B][nsplit][4][Nf]
    int64_t Nt, Nf;
    int64_t split_len;          // samples per split (multiple of UM_TS)
    int nsplit, nfb, nparts;
    int flush_ksteps;           // k-steps between drains of D_W
    float trunc_ulps;           // truncation compensation at each drain of D_W (tc_trunc_comp): < 0 the model, 0 off; pair form also > 0: ulps per k-step
    int unit_x;                 // 1: recA.x is a weight, not a measurement: no variance scaling, no V (second pass of the generalised periodogram)
    // short-grid form with the pre-pass fused in (accum_umma_small_kernel<..., FUSED_PRE>): steps 1-2 are done by each CTA itself
    // from the caller's arrays (short series: every CTA forms the mean and variance over the whole series, identically)
    const double* t; int64_t t_stride;      // series b at t + b * t_stride
    const float* x; int64_t x_stride;
    double f_min, df;
    double* part_var_out;       // [B]: sum (x - mean)^2, written by the series' first CTA for the finish step (nparts = 1)
    double* part_sum_out;       // [B]: sum x, likewise (refine_kernel takes the mean from it)
    u64* peak64; unsigned* counter;   // [B]: reset by the series' first CTA
};

// 1 / sigma as the fp32 factor applied to X before it is split into fp16 pairs (unit variance, so fp16
// neither overflows nor underflows).  The finish step recomputes the identical value (same fixed-order sum, same IEEE
// operations) to undo it exactly.
__device__ __forceinline__ float x_scale(const double* part_var, int nparts, int64_t Nt)
{
    double q = 0.0;
    for (int i = 0; i < nparts; ++i) q += part_var[i];
    const double var = q / (double)(Nt - 1);
    return (float)(1.0 / sqrt(var));
}

__device__ __forceinline__ unsigned pack_h2(float lo, float hi)
{
    const __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const unsigned*>(&h);
}
// Two fp32 -> packed fp16 pair rounded STOCHASTICALLY: the 13 bits `r` (< 2^13) go under the 10 mantissa bits fp16 keeps of fp32's 23, then
// round toward zero.  Unbiased: the rounding errors of an operand that hardly changes from sample to sample (e^{2ia} at low frequencies)
// no longer add up coherently in the one-pass sum D_V.  (fp16 subnormals are cut more coarsely than 13 bits: < 6e-8.)
__device__ __forceinline__ unsigned pack_h2_sr(float lo, float hi, unsigned r)
{
    unsigned d;
    asm("cvt.rz.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(__uint_as_float(__float_as_uint(hi) + r)), "f"(__uint_as_float(__float_as_uint(lo) + r)));
    return d;
}
__device__ __forceinline__ float2 unpack_h2(unsigned v)
{
    return __half22float2(*reinterpret_cast<const __half2*>(&v));
}
// step 3: signed 32-bit fixed-point turns -> radians in [-pi, pi) -> MUFU sin/cos, abs error ~2^-21
__device__ __forceinline__ void sincos_phase32(unsigned ph, float& c, float& s)
{
    const float ang = (float)(int)ph * LSP_RAD_PER_PHASE;
    c = __cosf(ang); s = __sinf(ang);
}
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
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
// 1-D bulk copy global -> shared (TMA without a tensor map), completion counted in bytes on `bar`
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
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
constexpr uint32_t umma_idesc(int M, int N) { return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24); }
// kind::f8f6f4: A format at bit 7, B format at bit 10; 1 = E5M2.
constexpr uint32_t UMMA_IDESC_E5M2 = (1u << 7) | (1u << 10);

// 32 lanes x N consecutive columns of fp32 accumulators -> N registers per thread (lane = TMEM lane).
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
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16])
{
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    #pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float (&v)[8])
{
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    #pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
// ------------------------------------------------------------------ truncation compensation of a drained accumulator
// How tcgen05.mma folds products into its fp32 accumulator, measured on B200 with one-element probes and with random operands
// against exact sums (round 2): the 16 (kind::f16) or 32 (kind::f8f6f4) products of an output element and
// the accumulator are aligned to the largest exponent among them with TWO extra bits, each truncated toward zero, summed, and
// the sum truncated toward zero to fp32 ((2^24 + 2) + 1 -> 2^24 + 2, - 0.5 -> 2^24, - 2^-10 -> unchanged, four times - 0.75 in
// one MMA -> 2^24).  In ulps of the RUNNING accumulator an MMA therefore loses, toward zero,
//     3/8 (the final truncation of a sum that carries two extra bits)  +  1/8 per product, signed by that product's own sign.
// For products of random sign (noise, and the small hi x lo cross terms of the correction MMAs) the second part averages out
// (measured: 0.19 ulp of the final value per MMA = 3/8 x the mean ratio rho of running to final ulp); for products that share
// the accumulator's sign (a coherent line) it adds 16/8 = 2 ulp per main MMA (measured: 1.06 - 1.14 ulp of the final value).
// The expected loss over a drain window of n k-steps, in ulps of its final value D_n, added back away from zero at the drain:
//     n x (c0 + 2 a) x rho(m) x ulp(D_n)
//   c0     3/8 per MMA that adds into the accumulator per k-step (0.75: main + e5m2 corrections; 1.125: main + two fp16 corrections);
//   a      the excess of the main MMA's products that share the accumulator's sign, P(p > 0) - P(p < 0), estimated from the window
//          itself: for products p ~ N(mu, s^2) it is erf(mu / (s sqrt 2)) ~ (2/pi) mu / E|p| with mu = |D_n| / (16 n), E|p| = E|X| E|cos|
//          = 0.51 for the unit-variance X of the tensor forms (0 for noise, whose sums grow like sqrt(n); -> 1 for a line in phase);
//          inv_coherent = (2/pi) / (16 n E|p|);
//   rho(m) = 1 - 2 / (3 m), m in [1, 2) the mantissa of D_n: a sum that grows from 0 to D_n -- linearly, or like a random walk with the
//          same conditional mean (t/n) D_n -- passes through the binades below its final one.
__device__ __forceinline__ float tc_trunc_comp(float v, float n_ksteps, float c0, float inv_coherent)
{
    const unsigned bits = __float_as_uint(v);
    const float ulp = __uint_as_float(bits & 0x7f800000u) * 1.1920929e-7f;          // 2^(e-23)
    const float rho = 1.f - __fdividef(0.6666667f, __uint_as_float((bits & 0x007fffffu) | 0x3f800000u));
    const float a = fminf(fabsf(v) * inv_coherent, 1.f);
    return v + copysignf(n_ksteps * fmaf(2.f, a, c0) * rho * ulp, v);
}
constexpr float TC_MEAN_ABS_PRODUCT = 0.508f;          // E|X| E|cos| for X ~ N(0, 1)
constexpr float TC_MEAN_ABS_COS = 0.637f;              // the weight pass of the generalised periodogram: X = 1

__device__ __forceinline__ void sts128(uint32_t saddr, unsigned a, unsigned b, unsigned c, unsigned d)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" :: "r"(saddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ------------------------------------------------------------------ cluster scope (CTA pairs, cta_group::2)
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// Arrive on the mbarrier at the same shared-memory offset in CTA `cta` of the cluster.  No .release.cluster: that
// lowers to MEMBAR.ALL.GPU (~1 us per stage on the critical path).  What the remote waiter goes on to read is this
// CTA's shared memory, read by the tensor core (async proxy); those writes were completed and made visible to the
// async proxy (fence.proxy.async / TMA complete_tx) before the local barrier this thread waited on flipped.
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar, uint32_t cta)
{
    asm volatile("{\n\t.reg .b32 ra;\n\tmapa.shared::cluster.u32 ra, %0, %1;\n\t"
                 "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}" :: "r"(bar), "r"(cta) : "memory");
}
__device__ __forceinline__ void tc_commit_pair(uint32_t bar)     // arrives on `bar` in BOTH CTAs when all earlier MMAs are done
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 :: "r"(bar), "h"((unsigned short)3) : "memory");
}
__device__ __forceinline__ void tc_mma_f16_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_mma_f8_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

}  // namespace lsp
