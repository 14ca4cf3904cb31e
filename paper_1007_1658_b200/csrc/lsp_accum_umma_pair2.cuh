// lsp_accum_umma_pair2.cuh -- the tcgen05 form of steps 3-5 for LONG grids: a CTA pair (cta_group::2) per 32,768
// frequencies, one operand streamed from a table, the other generated and shared by the pair (algebra: lsp_tc.cuh).
//
//     k = kb + 256 h + l,   l < 256 fine (table, M side),   h < 128 coarse (generated, N side),   kb = 32,768 * pair
//     theta_jk = [2 pi frac(u_j + (kb + 256 h) v_j)]  +  [2 pi frac(l v_j)]  =  a_jh + b_jl          (exact 64-bit turns, G3)
//     W[l,h] = sum_j e^{i b_jl} (X_j e^{i a_jh}),    V[l,h] = sum_j e^{2i b_jl} (e^{2i a_jh} / 2)     (eq. (8))
//
// The fine factor e^{i b_jl} depends on the sample and on l only -- NOT on the frequency block -- so a pre-pass
// (`umma_ftable_pair_kernel`) writes it ONCE per time chunk, already as the shared-memory image the tensor core reads
// (no-swizzle K-major core matrices; planes: fp16 (c, s), e5m2 [hi | lo], fp16 double angle; 2 x 12 KB per k-step of 8
// samples), and every CTA streams ITS 128 rows with one cp.async.bulk (TMA) per stage onto the stage's mbarrier; the
// table is read once per CTA pair, mostly from L2 (CTAs of one wave work on the same few time splits in lockstep).
// One tcgen05.mma.cta_group::2 of M = 256, N = 256: the M rows are the fine index l -- CTA r accumulates ITS 128 rows in
// ITS TMEM -- and the N columns (h,Re), (h,Im) are the generated operand, of which each CTA makes only HALF (64 coarse
// values h, both parts): 64 sin/cos pairs per sample per CTA.  The (h,Im) row is a permutation of the (h,Re) row
// ((xc, -xs) -> (xs, xc)): PRMT / LOP3 on the packed words, no extra arithmetic.  A stage-step (two k-steps) is
// 256 thread-tasks, so the 16 producer warps work as two groups of 8 on alternate stage-steps.  Per k-step:
//     D_W += T_hi G_hi (kind::f16);  D_W += T_8 G_8 (kind::f8f6f4, K = 32: both hi*lo corrections);  D_V += T_V G_V (kind::f16)
//
// TMEM (per CTA): lane = l - 128 r;  column n = 128 r' + 64 part + h',  h = 64 r' + h'  (r' = CTA that generated it);
// D_W in columns 0..255, D_V in 256..511.  For a fixed column the 32 lanes of a warp are 32 consecutive
// frequencies: the drain into `ws` is coalesced.
//
// Time chunks.  The table is 3 KB per sample, so the host bounds it (1 GiB by default): the series is cut into chunks,
// each with its own table pre-pass + accumulate launch on the same table buffer; later chunks fold into `ws`
// (`accumulate` = 1: the first drain read-modify-writes too).  Fixed order, no atomics: deterministic.
//
// Synchronisation (all mbarriers; s = stage):
//   FULL[s]   in each CTA, count 8 + 1 + tx: the 8 producer warps of the stage's group and the CTA's own cp.async.bulk.
//   PEER[s]   in CTA 0, count 1: CTA 1's otherwise idle MMA warp forwards "my FULL[s] completed" by a remote arrive;
//             the issuing thread of CTA 0 waits FULL[s] and PEER[s].
//   EMPTY[s]  in each CTA, count 1: tcgen05.commit.cta_group::2 multicast to both CTAs frees the stage in both.
//   ACCF      in each CTA, count 1 (commit multicast): every MMA so far has completed, drain may read TMEM.
//   ACCE      in CTA 0, count 32: the 16 drain warps of each CTA (CTA 1's by remote arrive) have read D_W.
#pragma once
#include "lsp_tc.cuh"

namespace lsp {

constexpr int UM_GEN_WARPS = 16;                                  // producer (and drain) warps per CTA; warp 16 issues the MMAs
constexpr int UP_B_HALF = 128 * 32;                               // one table plane of a k-step in ONE CTA: 128 rows x 32 bytes
constexpr int UP_GROUP_BYTES = 3 * UP_B_HALF;                     // per k-step per CTA: T_hi, T_8, T_V (12 KB)
constexpr int U2_TABLE_BYTES_PER_KSTEP = 2 * UP_GROUP_BYTES;      // both CTAs of the pair: 24 KB per 8 samples = 3 KB per sample
constexpr int U2_TABLE_PAD_KSTEPS = 2;                            // the last stage's bulk copy may read one k-step past the data
// M = 256 (both CTAs), N = 256, fp32 accumulate; kind::f16 and kind::f8f6f4 (e5m2 x e5m2)
constexpr uint32_t UP_IDESC = umma_idesc(256, 256);
constexpr uint32_t UP_IDESC_F8 = UP_IDESC | UMMA_IDESC_E5M2;

struct UmmaPairParams {
    UmmaParams u;                   // u.nfb = 2 * npairs; u.split_len / u.nsplit divide the CHUNK; u.Nt = samples of the whole series
    const unsigned char* btable;    // [B or 1][2][ngroups][UP_GROUP_BYTES] for the chunk's samples
    int64_t half_stride;            // bytes between the two 128-row halves of one series' table
    int64_t table_stride;           // bytes between the tables of consecutive series (0: shared times)
    int64_t j0, chunk_len;          // the chunk: samples j0 .. j0 + chunk_len - 1
    int nsplit_grid;                // time splits this launch covers (a short last chunk has fewer than u.nsplit, the stride of `ws`)
    int accumulate;                 // 1: `ws` holds the sums of earlier chunks
    const float4* recW;             // weighted generalised periodogram: recW[j].x = sqrt of the normalised weight w_j (and u.recA.x carries one
                                    // factor sqrt(w_j) already, lsp_prepass.cuh): X = recA.x recW.x, and V = sum w e^{2i theta}; else NULL
};

constexpr int U2_FPP = 256 * UM_H;                                // frequencies per CTA pair
constexpr int U2_HC = 64;                                         // coarse values generated per CTA
#ifndef LSP_U2_KPS
#define LSP_U2_KPS 2
#endif
constexpr int U2_KPS = LSP_U2_KPS;                                // k-steps per ring stage.  Measured on C3 / C5 (accumulate ms): 1 -> 2.01 / 22.1
                                                                  // (a wait + commit per three MMAs costs more than the finer hand-over gains),
                                                                  // 2 -> 1.64 / 17.0 (default), 4 -> 1.62 / 16.9 (needs a longer table tail; not adopted)
static_assert(U2_KPS == 1 || U2_KPS == 2, "the table is padded for stages of at most two k-steps");
constexpr int U2_STAGES = 8 / U2_KPS;                             // the ring always holds 8 k-steps
constexpr int U2_GSLOT = U2_KPS * 3 * UM_A_BYTES;                 // generated planes of one stage
constexpr int U2_STAGE_BYTES = U2_GSLOT + U2_KPS * UP_GROUP_BYTES; // + this CTA's table rows
constexpr int U2_GT = 128 * U2_KPS;                               // thread-tasks per stage-step = threads of a producer group
#ifndef LSP_U2_GROUPS
#define LSP_U2_GROUPS (512 / (128 * LSP_U2_KPS))
#endif
constexpr int U2_GROUPS = LSP_U2_GROUPS;                          // producer groups: group g owns the stage-steps it = g (mod U2_GROUPS)
constexpr int U2_GROUP_WARPS = U2_GT / 32;
constexpr int U2_PROD_WARPS = U2_GROUPS * U2_GROUP_WARPS;         // 16; they also drain; warp 16 issues the MMAs
constexpr int U2_THREADS = (U2_PROD_WARPS + 1) * 32;
constexpr int U2_TILE_STEPS = (UM_TS / UM_KS) / U2_KPS;           // stage-steps per 128-sample record tile
constexpr int U2_REC_BYTES = U2_GROUPS * 2 * UM_TS * 16;          // [group][buffer][128 samples] records
constexpr size_t U2_SMEM = (size_t)U2_STAGES * U2_STAGE_BYTES + U2_REC_BYTES + 256;

// ------------------------------------------------------------------ pre-pass: the fine-operand table
// table[r][g][plane][chunk][l & 127][16 bytes], r = l >> 7: plane 0 = (c, s) fp16, 1 = [e5m2(c_h, s_h) | e5m2(c - c_h, s - s_h)],
// 2 = (cos 2b, sin 2b) fp16; b = 2 pi frac(l v_j).  grid (ngroups, series), 512 threads = 2 K-chunks x 256 fine indices;
// group g holds samples j0 + 8g .. j0 + 8g + 7 of the chunk [j0, j1).
__device__ __forceinline__ unsigned u2_hash(unsigned x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}
__global__ void __launch_bounds__(512) umma_ftable_pair_kernel(const ulonglong2* __restrict__ recB, int64_t j0, int64_t j1, int64_t rec_stride,
                                                               unsigned char* __restrict__ table, int64_t half_stride, int64_t table_stride, int corr16)
{
    const int64_t g = blockIdx.x;
    const unsigned l = threadIdx.x & 255u, chunk = threadIdx.x >> 8;
    const ulonglong2* rb = recB + (int64_t)blockIdx.y * rec_stride;
    unsigned hh[4], h8[4], l8[4], vv[4], l16[4];
    #pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int64_t j = j0 + g * UM_KS + chunk * 4 + i;
        const u64 v = (j < j1) ? __ldg(&rb[j].y) : 0ull;                // beyond the chunk: e^{i0}; the generated operand is zero there
        const unsigned v32 = (unsigned)((v + 0x80000000ull) >> 32);
        float c, s;
        sincos_phase32(l * v32, c, s);
        hh[i] = pack_h2(c, s);
        const float2 hf = unpack_h2(hh[i]);
        h8[i] = pack_e5m2_h2(hh[i]);
        l8[i] = pack_e5m2(c - hf.x, s - hf.y);
        l16[i] = pack_h2(c - hf.x, s - hf.y);
        const float cc = c + c;
        // e^{2ib} to fp16 by STOCHASTIC rounding (13 pseudo-random bits under the fp16 mantissa, then truncation).  D_V has one fp16 pass, and
        // where b hardly moves over the series (l df T << 1: the low frequencies) round-to-nearest makes the SAME error in every sample --
        // cos 2b within one or two fp16 steps of 1 -- which sums coherently: |dV| = 2.8e-5 Nt at f T = 0.54 on the probe of DESIGN.md section 8,
        // i.e. 5e-5 ... 7e-5 of P_k on ANY series.  Unbiased rounding makes the errors independent: 5e-7 Nt there.  Deterministic (a hash of
        // the sample and fine index).
        const unsigned rb = u2_hash((unsigned)(j0 + g * UM_KS + chunk * 4 + i) * 256u + l);
        vv[i] = pack_h2_sr(fmaf(cc, c, -1.f), cc * s, rb & 0x1fffu);
    }
    unsigned char* base = table + (int64_t)blockIdx.y * table_stride + (int64_t)(l >> 7) * half_stride + g * (int64_t)UP_GROUP_BYTES;
    uint4* o = reinterpret_cast<uint4*>(base);
    constexpr int PLANE = UP_B_HALF / 16;
    const int row = (int)(chunk * (PLANE / 2) + (l & 127u));
    o[row] = make_uint4(hh[0], hh[1], hh[2], hh[3]);
    if (corr16) o[PLANE + row] = make_uint4(l16[0], l16[1], l16[2], l16[3]);      // plane 1 = fp16 (c - c_h, s - s_h)
    else o[PLANE + row] = make_uint4(h8[0] | (h8[1] << 16), h8[2] | (h8[3] << 16), l8[0] | (l8[1] << 16), l8[2] | (l8[3] << 16));
    o[2 * PLANE + row] = make_uint4(vv[0], vv[1], vv[2], vv[3]);
}

// ------------------------------------------------------------------ step 3: the generated (coarse) operand
// One task: coarse value h, 4 samples starting at rec[s0]: writes the 16-byte chunks of rows (h,Re) and (h,Im)
// (64 rows = 1,024 bytes apart) of the planes G_hi, G_8 = [e5m2(G_lo) | e5m2(G_hi)], G_V.  sG = address of row (h,Re).
__device__ __forceinline__ unsigned swap_halves(unsigned x) { return __byte_perm(x, 0u, 0x1032); }
__device__ __forceinline__ unsigned swap_bytes16(unsigned x) { return __byte_perm(x, 0u, 0x2301); }

template <bool TAIL, bool WEIGHTED, bool CORR16>
__device__ __forceinline__ void u2_gen(const float4* rec, int s0, unsigned h, uint32_t sG, int nvalid)
{
    unsigned hi[4], lo[4], h8[4], vv[4];
    #pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float4 r = rec[s0 + i];                                   // {X / sigma, pA32, w32, weight}: broadcast read
        float c, s;
        sincos_phase32(__float_as_uint(r.y) + h * __float_as_uint(r.z), c, s);
        const u64 cs = pack2(c, s);
        float xc, xs;
        unpack2(mul2(pack2(r.x, r.x), cs), xc, xs);
        hi[i] = pack_h2(xc, xs);
        const float2 hf = unpack_h2(hi[i]);
        float lc, ls;
        unpack2(fma2(pack2(hf.x, hf.y), pack2(-1.f, -1.f), pack2(xc, xs)), lc, ls);
        if (CORR16) lo[i] = pack_h2(lc, ls);
        else { lo[i] = pack_e5m2(lc, ls); h8[i] = pack_e5m2_h2(hi[i]); }
        float v0, v1;
        unpack2(fma2(pack2(c, c), cs, pack2(-0.5f, 0.f)), v0, v1);      // (cos^2 a - 1/2, cos a sin a) = e^{2ia} / 2
        if (WEIGHTED) { v0 *= r.w; v1 *= r.w; }                         // V = sum_j w_j e^{2i theta}
        vv[i] = pack_h2(v0, v1);                                        // (rounded stochastically like the table's plane: measured no gain, +1 %)
        if (TAIL && i >= nvalid) vv[i] = 0u;                            // pads (X = 0) must not count in V either
    }
    unsigned q0 = 0u, q1 = 0u, q2 = 0u, q3 = 0u;
    if (!CORR16) { q0 = lo[0] | (lo[1] << 16); q1 = lo[2] | (lo[3] << 16); q2 = h8[0] | (h8[1] << 16); q3 = h8[2] | (h8[3] << 16); }
    constexpr uint32_t IM = U2_HC * 16;                                 // row (h,Im) is 64 rows below row (h,Re)
    // row (h,Re) = (xc, -xs): flip the sign of the second component;  row (h,Im) = (xs, xc): swap the components
    sts128(sG, hi[0] ^ 0x80000000u, hi[1] ^ 0x80000000u, hi[2] ^ 0x80000000u, hi[3] ^ 0x80000000u);
    sts128(sG + IM, swap_halves(hi[0]), swap_halves(hi[1]), swap_halves(hi[2]), swap_halves(hi[3]));
    if (CORR16) {                                                       // plane 1 = G_lo in fp16, rows built as those of G_hi
        sts128(sG + UM_A_BYTES, lo[0] ^ 0x80000000u, lo[1] ^ 0x80000000u, lo[2] ^ 0x80000000u, lo[3] ^ 0x80000000u);
        sts128(sG + UM_A_BYTES + IM, swap_halves(lo[0]), swap_halves(lo[1]), swap_halves(lo[2]), swap_halves(lo[3]));
    } else {
    sts128(sG + UM_A_BYTES, q0 ^ 0x80008000u, q1 ^ 0x80008000u, q2 ^ 0x80008000u, q3 ^ 0x80008000u);
    sts128(sG + UM_A_BYTES + IM, swap_bytes16(q0), swap_bytes16(q1), swap_bytes16(q2), swap_bytes16(q3));
    }
    sts128(sG + 2 * UM_A_BYTES, vv[0] ^ 0x80000000u, vv[1] ^ 0x80000000u, vv[2] ^ 0x80000000u, vv[3] ^ 0x80000000u);
    sts128(sG + 2 * UM_A_BYTES + IM, swap_halves(vv[0]), swap_halves(vv[1]), swap_halves(vv[2]), swap_halves(vv[3]));
}

// ------------------------------------------------------------------ step 5: drain 64 accumulator columns into ws
// Thread = TMEM lane = fine index; its 64 registers are 64 consecutive coarse values h (frequency stride 256).
//
// Truncation compensation: tc_trunc_comp (lsp_tc.cuh).  mode < 0 (default): the model; mode > 0: that many ulps of D_n per k-step,
// whatever the data (ablation, LSP_PARAM_TRUNC); mode = 0: nothing is added.
__device__ __forceinline__ void u2_drain64(uint32_t taddr, float* dst, int64_t k0, int64_t Nf, bool first, float mode, float n_ksteps, float c0, float inv_coherent)
{
    #pragma unroll 1
    for (int half = 0; half < 2; ++half) {
        float v[32];
        tmem_ld32(taddr + 32u * half, v);
        if (mode != 0.f) {
            #pragma unroll
            for (int i = 0; i < 32; ++i) {
                if (mode < 0.f) v[i] = tc_trunc_comp(v[i], n_ksteps, c0, inv_coherent);
                else v[i] += copysignf(n_ksteps * mode * __uint_as_float(__float_as_uint(v[i]) & 0x7f800000u) * 1.1920929e-7f, v[i]);
            }
        }
        const int64_t kh = k0 + (int64_t)half * 32 * 256;
        if (!first) {
            #pragma unroll
            for (int i = 0; i < 32; ++i) { const int64_t k = kh + (int64_t)i * 256; if (k < Nf) v[i] += dst[k]; }
        }
        #pragma unroll
        for (int i = 0; i < 32; ++i) { const int64_t k = kh + (int64_t)i * 256; if (k < Nf) dst[k] = v[i]; }
    }
}

// ------------------------------------------------------------------ the kernel
// grid.x = B * nsplit * (2 * npairs) (CTA of the pair fastest, then the pair), clusters of 2, U2_THREADS threads,
// U2_SMEM bytes of dynamic shared memory, one CTA per SM.  q.u.nfb = 2 * npairs, npairs = ceil(Nf / 32,768).
// CORR16 (LSP_PARAM_CORR = 1): plane 1 of both operands holds fp16 lo parts and the corrections are two kind::f16 MMAs.
template <bool CORR16>
__global__ void __launch_bounds__(U2_THREADS, 1) accum_umma_pair2_kernel(const UmmaPairParams q)
{
    const UmmaParams& p = q.u;
    extern __shared__ __align__(128) unsigned char um_smem[];
    float4* rec_all = reinterpret_cast<float4*>(um_smem + U2_STAGES * U2_STAGE_BYTES);            // [group][2][UM_TS] {X/sigma, pA32, w32, -}
    uint64_t* bars = reinterpret_cast<uint64_t*>(um_smem + U2_STAGES * U2_STAGE_BYTES + U2_REC_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * U2_STAGES + 2);

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % q.nsplit_grid);
    const int64_t b = unit / q.nsplit_grid;
    const int64_t kb = (int64_t)(fb >> 1) * U2_FPP;
    const int64_t j_begin = q.j0 + (int64_t)sp * p.split_len;
    const int64_t j_end = min(q.j0 + q.chunk_len, j_begin + p.split_len);
    const int n_samp = (int)(j_end - j_begin);                          // split_len < 2^31
    const int nks = (n_samp + UM_KS - 1) / UM_KS;
    const int nst = (nks + U2_KPS - 1) / U2_KPS;                        // stage-steps (two k-steps each)
    const int flush_st = max(U2_GROUPS, (p.flush_ksteps / U2_KPS) / U2_GROUPS * U2_GROUPS);   // a multiple of the group count: every group sees the same windows
    const int nwin = (nst + flush_st - 1) / flush_st;

    const uint32_t s_stage = smem_u32(um_smem), s_bar = smem_u32(bars);
    const uint32_t bar_accf = s_bar + 8u * (3 * U2_STAGES), bar_acce = bar_accf + 8u;
#define U2_FULL(s) (s_bar + 8u * (unsigned)(s))
#define U2_EMPTY(s) (s_bar + 8u * (unsigned)(U2_STAGES + (s)))
#define U2_PEER(s) (s_bar + 8u * (unsigned)(2 * U2_STAGES + (s)))

    if (tid == 0) {
        for (int s = 0; s < U2_STAGES; ++s) { mbar_init(U2_FULL(s), U2_GROUP_WARPS + 1); mbar_init(U2_EMPTY(s), 1); mbar_init(U2_PEER(s), 1); }
        mbar_init(bar_accf, 1);
        mbar_init(bar_acce, 2 * UM_GEN_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster_sync_all();
    if (w == U2_PROD_WARPS) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"((uint32_t)UM_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);
    cluster_sync_all();

    if (w < U2_PROD_WARPS) {
        // ===================== producers: generated operand (step 3), TMA of this CTA's table rows, drain (step 5) =====================
        const unsigned grp = w / U2_GROUP_WARPS, tg = tid & (unsigned)(U2_GT - 1);                   // group `grp` owns the stage-steps it = grp (mod 2)
        float4* rec = rec_all + grp * (2 * UM_TS);
        const float4* recA = p.recA + b * p.Nt;
        const ulonglong2* recB = p.recB + b * p.Nt;
        const unsigned char* tab = q.btable + b * q.table_stride + (int64_t)rank * q.half_stride + ((j_begin - q.j0) / UM_KS) * (int64_t)UP_GROUP_BYTES;
        const float xs = (tg < UM_TS) ? (p.unit_x ? 1.f : x_scale(p.part_var + b * p.nparts, p.nparts, p.Nt)) : 0.f;
        const bool weighted = q.recW != nullptr;
        const float4* recW = weighted ? q.recW + b * p.Nt : nullptr;
        float pre_x = 0.f, pre_w = 1.f; u64 pre_u = 0ull, pre_v = 0ull; bool pre_ok = false;
        auto prefetch = [&](int ti) {
            const int64_t j = j_begin + (int64_t)ti * UM_TS + tg;
            pre_ok = (tg < UM_TS) && (j < j_end);
            if (pre_ok) {
                pre_x = __ldg(&recA[j].x); const ulonglong2 r = __ldg(recB + j); pre_u = r.x; pre_v = r.y;
                if (weighted) pre_w = __ldg(&recW[j].x);
            }
        };
        prefetch(0);
        const unsigned hl = tg & 63u, h = (unsigned)U2_HC * rank + hl;   // coarse value: local row, global index
        const int chunk = (int)((tg >> 6) & 1u), kk = (int)(tg >> 7);    // 4 samples `chunk` of k-step `kk` of the stage
        const uint32_t g_off = (uint32_t)kk * (3 * UM_A_BYTES) + (uint32_t)chunk * (UM_A_BYTES / 2) + hl * 16u;
        const int samp_off = kk * UM_KS + chunk * 4;                     // first sample of the task within the stage-step
        // drain role: TMEM lane quadrant q4, column group cg = (generating CTA r', part)
        const unsigned q4 = w & 3u, cg = w >> 2;
        float* ws_unit = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
        const int64_t k0 = kb + (int64_t)256 * (U2_HC * (cg >> 1)) + (int64_t)(128u * rank + 32u * q4 + lane);
        const uint32_t t_drain = tmem + ((32u * q4) << 16) + 64u * cg;
        int ti_cur = -1;

        for (int f = 0; f < nwin; ++f) {
            const int it_end = min(nst, (f + 1) * flush_st);
            const int it0 = f * flush_st;
            for (int it = it0 + ((int)grp + U2_GROUPS - it0 % U2_GROUPS) % U2_GROUPS; it < it_end; it += U2_GROUPS) {
                const int s = it & (U2_STAGES - 1);
                const uint32_t ph = (uint32_t)(it / U2_STAGES) & 1u;
                const int ti = it / U2_TILE_STEPS;                      // stage-steps per record tile
                if (ti != ti_cur) {                                     // next record tile of this group (buffer ti & 1)
                    ti_cur = ti;
                    if (tg < UM_TS) {
                        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);     // pad: X = 0, phases 0
                        if (pre_ok) {
                            const u64 pa = pre_u + (u64)kb * pre_v;     // u + kb v (mod 1, 64-bit wrap; reading G3)
                            r.x = pre_x * xs * pre_w;                   // (pre_w = 1 without weights)
                            r.y = __uint_as_float((unsigned)((pa + 0x80000000ull) >> 32));
                            r.z = __uint_as_float((unsigned)((256ull * pre_v + 0x80000000ull) >> 32));
                            r.w = pre_w * pre_w;
                        }
                        rec[(ti & 1) * UM_TS + tg] = r;
                        prefetch(ti + 1);
                    }
                    asm volatile("bar.sync %0, %1;" :: "r"(1u + grp), "n"(U2_GT) : "memory");
                }
                mbar_wait(U2_EMPTY(s), ph ^ 1u);                        // the pair's MMAs that read this stage have completed
                const uint32_t st = s_stage + (uint32_t)s * U2_STAGE_BYTES;
                if (tg < 32u) {                                         // warp-uniform: only the group's first warp runs the copy-issue code
                    if (lane == 0) {                                    // this CTA's 128 table rows of the two k-steps: one bulk copy
#ifdef LSP_U2_DBG_NOTMA
                        mbar_arrive(U2_FULL(s));
#else
                        mbar_expect_tx(U2_FULL(s), U2_KPS * UP_GROUP_BYTES);
                        tma_bulk_g2s(st + U2_GSLOT, tab + (int64_t)it * (U2_KPS * UP_GROUP_BYTES), U2_KPS * UP_GROUP_BYTES, U2_FULL(s));
#endif
                    }
                    __syncwarp();
                }
                const int s0 = (it % U2_TILE_STEPS) * (U2_KPS * UM_KS) + samp_off;  // within the 128-sample record tile
                const int left = n_samp - (it * (U2_KPS * UM_KS) + samp_off);
#ifndef LSP_U2_DBG_NOGEN
                if (!weighted) {
                    if (left >= 4) u2_gen<false, false, CORR16>(rec + (ti & 1) * UM_TS, s0, h, st + g_off, 4);      // `left` is warp-uniform
                    else u2_gen<true, false, CORR16>(rec + (ti & 1) * UM_TS, s0, h, st + g_off, max(0, left));
                } else {
                    if (left >= 4) u2_gen<false, true, CORR16>(rec + (ti & 1) * UM_TS, s0, h, st + g_off, 4);
                    else u2_gen<true, true, CORR16>(rec + (ti & 1) * UM_TS, s0, h, st + g_off, max(0, left));
                }
#else
                (void)s0; (void)left; (void)h; (void)g_off;
#endif
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(U2_FULL(s));
            }
            // ---- drain window f (warps 0..15 of both CTAs)
            if (w >= UM_GEN_WARPS) continue;
            const bool last = (f == nwin - 1);
            mbar_wait(bar_accf, (uint32_t)f & 1u);
            tc_fence_after();
            {
                const float nk = (float)((it_end - f * flush_st) * U2_KPS);                 // k-steps of this window
                const float mean_abs_product = p.unit_x ? TC_MEAN_ABS_COS : TC_MEAN_ABS_PRODUCT;
                u2_drain64(t_drain, ws_unit + (int64_t)(cg & 1u) * p.Nf, k0, p.Nf, f == 0 && !q.accumulate, p.trunc_ulps, nk,
                           CORR16 ? 1.125f : 0.75f, 0.6366198f / (16.f * nk * mean_abs_product));
            }
            // D_V is drained with D_W (round 2): left to accumulate over the whole split it lost ~n ulp toward zero wherever sum e^{2i theta}
            // is coherent (f T < ~1, aliases of regular sampling, any series with a trend), an error that grew with the split length and
            // that Nt / (Nt - R) amplifies (found by a randomised sweep on series with a drift: up to 1e-3 of max P)
            if (!p.unit_x) u2_drain64(t_drain + 256u, ws_unit + (int64_t)(2 + (cg & 1u)) * p.Nf, k0, p.Nf, f == 0 && !q.accumulate, 0.f, 0.f, 0.f, 0.f);
            (void)last;
            tc_fence_before();
            __syncwarp();
            if (lane == 0) { if (rank == 0) mbar_arrive(bar_acce); else mbar_arrive_remote(bar_acce, 0u); }
        }
    } else if (lane == 0 && rank == 0) {
        // ===================== step 4: the single MMA-issuing thread of the pair =====================
        int f = 0;
        for (int it = 0; it < nst; ++it) {
            const int s = it & (U2_STAGES - 1);
            const uint32_t ph = (uint32_t)(it / U2_STAGES) & 1u;
            mbar_wait(U2_FULL(s), ph);
            mbar_wait(U2_PEER(s), ph);
            tc_fence_after();
            const bool win_first = (it == f * flush_st);
            #pragma unroll
            for (int kk = 0; kk < U2_KPS; ++kk) {
                const uint32_t g0 = s_stage + (uint32_t)s * U2_STAGE_BYTES + kk * (3 * UM_A_BYTES);           // generated: N side
                const uint32_t t0 = s_stage + (uint32_t)s * U2_STAGE_BYTES + U2_GSLOT + kk * UP_GROUP_BYTES; // table: M side
                const uint64_t dGh = umma_desc(g0, UM_A_BYTES / 2, 128), dG8 = umma_desc(g0 + UM_A_BYTES, UM_A_BYTES / 2, 128);
                const uint64_t dGv = umma_desc(g0 + 2 * UM_A_BYTES, UM_A_BYTES / 2, 128);
                const uint64_t dTh = umma_desc(t0, UP_B_HALF / 2, 128), dT8 = umma_desc(t0 + UP_B_HALF, UP_B_HALF / 2, 128);
                const uint64_t dTv = umma_desc(t0 + 2 * UP_B_HALF, UP_B_HALF / 2, 128);
#ifndef LSP_U2_DBG_NOMMA
                tc_mma_f16_pair(tmem, dTh, dGh, UP_IDESC, (!win_first || kk > 0) ? 1u : 0u);
                if (CORR16) {                                           // plane 1 holds fp16 lo parts: A_lo B_hi + A_hi B_lo as two fp16 MMAs
                    tc_mma_f16_pair(tmem, dT8, dGh, UP_IDESC, 1u);
                    tc_mma_f16_pair(tmem, dTh, dG8, UP_IDESC, 1u);
                } else tc_mma_f8_pair(tmem, dT8, dG8, UP_IDESC_F8, 1u);
                if (!p.unit_x)                                          // (the unit-weight pass of the generalised periodogram needs no V: CC, CS come from the first pass)
                    tc_mma_f16_pair(tmem + 256u, dTv, dGv, UP_IDESC, (!win_first || kk > 0) ? 1u : 0u);
#else
                (void)dTh; (void)dGh; (void)dT8; (void)dG8; (void)dTv; (void)dGv; (void)win_first;
#endif
            }
            tc_commit_pair(U2_EMPTY(s));
            const bool last = (it == nst - 1);
            if (it + 1 == (f + 1) * flush_st || last) {
                tc_commit_pair(bar_accf);
                if (!last) { mbar_wait(bar_acce, (uint32_t)f & 1u); tc_fence_after(); }
                ++f;
            }
        }
    } else if (lane == 0) {
        // ===================== CTA 1: forward "my stage is full" to the issuing thread in CTA 0 =====================
        for (int it = 0; it < nst; ++it) {
            const int s = it & (U2_STAGES - 1);
            const uint32_t ph = (uint32_t)(it / U2_STAGES) & 1u;
            mbar_wait(U2_FULL(s), ph);
            mbar_arrive_remote(U2_PEER(s), 0u);
        }
    }
#undef U2_FULL
#undef U2_EMPTY
#undef U2_PEER

    __syncwarp();
    tc_fence_before();
    cluster_sync_all();
    if (w == U2_PROD_WARPS) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((uint32_t)UM_TMEM_COLS) : "memory");
    }
}

}  // namespace lsp
