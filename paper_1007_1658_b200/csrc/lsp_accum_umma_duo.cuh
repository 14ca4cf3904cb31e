// lsp_accum_umma_duo.cuh -- the tcgen05 form of steps 3-5 for BATCHES of short series: two series per CTA.
//
// accum_umma_small_kernel<16> gives one series 128 fine x 16 coarse = 2,048 frequencies and is bound by operand
// generation: 128 + 16 = 144 MUFU sin/cos pairs per sample for 2,048 terms.  The balanced split 64 x 32 needs only 96,
// but an MMA has M = 128 rows.  Here the 128 rows are TWO series x 64 fine values, and the N = 128 columns are two
// series x (32 coarse values) x (Re, Im):
//     A[(s,h)][j] = X_sj e^{i a_sjh},   B[(s',l,part)][j] = e^{i b_s'jl},   k = kb + 64 l + h,
//     a_sjh = 2 pi frac(u_sj + (kb + h) v_sj),  b_sjl = 2 pi frac(64 l v_sj)           (exact 64-bit turns, reading G3)
// The K index is the sample number j, which both series of a batch share (same Nt), so the diagonal blocks s = s' of
//     D[(s,h)][(s',l,part)] = sum_j A[(s,h)][j] B[(s',l,part)][j]
// are the sums of eq. (8) of series s; the off-diagonal blocks (series s against the times of
// series s') are computed by the tensor core and never read -- the tensor pipe is far from busy here.
// Per pair of samples 2 x 64 + 2 x 32 = 192 sin/cos pairs = 96 per series instead of 144.
// Operand precision (fp16 hi + lo, three products for W, one for V), the stage ring, the periodic drain of D_W and
// the layout of `ws` are those of lsp_accum_umma_small.cuh; D_W: TMEM columns 0..127, D_V: 128..255; two CTAs per SM.
#pragma once
#include "lsp_accum_umma_small.cuh"
#include "lsp_refine.cuh"

namespace lsp {

constexpr int UD_H = 64;                                // fine values per series
constexpr int UD_L = 32;                                // coarse values per series
constexpr int UD_FPB = UD_H * UD_L;                     // frequencies per series per CTA
constexpr int UD_STAGES = 4;
constexpr int UD_STAGE_BYTES = 6 * UM_A_BYTES;          // A_hi, A_lo, A_V, B_hi, B_lo, B_V: 128 rows x 32 bytes each
constexpr int UD_REC_BYTES = 2 * 2 * UM_TS * 16;        // [series][buffer][128 samples]
constexpr int UD_RECW_BYTES = 2 * UM_RECW_BYTES;        // ... and their normalised weights (weighted generalised periodogram)
constexpr size_t UD_SMEM = (size_t)UD_STAGES * UD_STAGE_BYTES + UD_REC_BYTES + UD_RECW_BYTES + 256;
constexpr int UD_TMEM_COLS = 256;
constexpr uint32_t UD_IDESC = umma_idesc(UM_H, 128);   // M = 128, N = 128

// One B task: series s, coarse value l, 4 samples: rows (s,Re,l) and (s,Im,l) of B_hi, B_lo, B_V.  sB = address of row (s,Re,l).
__device__ __forceinline__ void ud_gen_b(const float4* rec, int s0, unsigned l, uint32_t sB)
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
    constexpr uint32_t IM = UD_L * 16;                                  // row (s,Im,l) is 32 rows below row (s,Re,l)
    sts128(sB, rh[0], rh[1], rh[2], rh[3]);
    sts128(sB + IM, ih[0], ih[1], ih[2], ih[3]);
    sts128(sB + UM_A_BYTES, rl[0], rl[1], rl[2], rl[3]);
    sts128(sB + UM_A_BYTES + IM, il[0], il[1], il[2], il[3]);
    sts128(sB + 2 * UM_A_BYTES, rv[0], rv[1], rv[2], rv[3]);
    sts128(sB + 2 * UM_A_BYTES + IM, iv[0], iv[1], iv[2], iv[3]);
}

// Drain 32 accumulator columns (one series, one of Re / Im) of this warp's 32 TMEM lanes into one plane of ws:
// thread = lane = fine value h, column l is frequency k0 + 64 l (coalesced over the lanes).
// n_ksteps > 0: D_W of a drain window of that many k-steps: the expected truncation loss is added back (tc_trunc_comp, three fp16 MMAs).
__device__ __forceinline__ void ud_drain(uint32_t taddr, float* dst, int64_t k0, int64_t Nf, bool first, bool live, float n_ksteps = 0.f, float inv_coherent = 0.f)
{
    #pragma unroll 1
    for (int part = 0; part < 2; ++part) {
        float v[16];
        tmem_ld16(taddr + 16u * part, v);
        if (!live) continue;
        if (n_ksteps > 0.f) {
            #pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = tc_trunc_comp(v[i], n_ksteps, 1.125f, inv_coherent);
        }
        const int64_t kp = k0 + (int64_t)part * 16 * UD_H;
        if (!first) {
            #pragma unroll
            for (int i = 0; i < 16; ++i) { const int64_t k = kp + (int64_t)i * UD_H; if (k < Nf) v[i] += dst[k]; }
        }
        #pragma unroll
        for (int i = 0; i < 16; ++i) { const int64_t k = kp + (int64_t)i * UD_H; if (k < Nf) dst[k] = v[i]; }
    }
}

struct UmmaDuoParams {
    UmmaParams u;                   // u.nfb = ceil(Nf / 2,048)
    int64_t B;                      // series in the batch; the CTA's second series may not exist (odd B)
    // fused steps 6-7: when one CTA sees ALL samples of its series in one drain window (nsplit = 1, Nt <= the drain interval)
    // its accumulators are the sums of eq. (8), and every thread holds XC, XS, CC - n/2, CS of its frequencies.
    int fuse;
    float* P; int64_t p_stride;     // nullable
    int32_t* peak_idx; float* peak_val; u64* peak64; unsigned* counter;   // nullable (all or none)
    RefineList list;                // fused epilogue: where the ill-conditioned frequencies go (lsp_refine.cuh); head NULL: nowhere
    float refine_r2;                //   ... those with R^2 above this (refine_amplification); +inf: none
};

// Steps 6-7 in the epilogue (same arithmetic as finish_kernel, eqs (5)-(7) PAPER.md:61-70 over the common denominator):
// thread = fine value h of series `db`; 16 coarse values l0..l0+15 -> frequencies kb + 64 l + h.
__device__ __forceinline__ void ud_finish16(const UmmaDuoParams& q, uint32_t tbase, int64_t db, bool live, int64_t kh, unsigned l0, unsigned lane)
{
    const UmmaParams& p = q.u;
    u64 best = 0ull;
    double inv2var = 0.0;
    const double Nt = (double)p.Nt;
    const float Nt_f = (float)p.Nt;
    if (live) {
        double qv = 0.0;
        for (int i = 0; i < p.nparts; ++i) qv += p.part_var[db * p.nparts + i];
        double var = qv / (double)(p.Nt - 1);                           // sample variance (reading G1)
        const double sc = (double)(float)(1.0 / sqrt(var));             // X was scaled by the fp32 x_scale(): undo it exactly
        var *= sc * sc;
        inv2var = 0.5 / var;
    }
    #pragma unroll 1
    for (unsigned c8 = 0; c8 < 16; c8 += 8) {
        float xc[8], xs[8], cc[8], cs[8];
        tmem_ld8(tbase + c8, xc);
        tmem_ld8(tbase + c8 + (uint32_t)UD_L, xs);
        tmem_ld8(tbase + c8 + 128u, cc);
        tmem_ld8(tbase + c8 + 128u + (uint32_t)UD_L, cs);
        if (!live) continue;
        const float inv2var_f = (float)inv2var;
        const float redo_r2 = fminf(0.25f * Nt_f * Nt_f, q.refine_r2);
        // fp32 where R <= Nt/2 (no amplification of the rounding of S Nt - D R); fp64 where the denominator Nt^2 - R^2 gets small
        float pf[8];
        #pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float A = 2.f * cc[i], Bv = 2.f * cs[i], R2 = fmaf(A, A, Bv * Bv);
            const float xc2 = xc[i] * xc[i], xs2 = xs[i] * xs[i], S = xc2 + xs2;
            const float DR = fmaf(xc2 - xs2, A, 2.f * xc[i] * xs[i] * Bv);
            pf[i] = fmaxf(2.f * fmaf(S, Nt_f, -DR), 0.f) / fmaf(Nt_f, Nt_f, -R2) * inv2var_f;
            if (R2 > redo_r2) {
                // ill-conditioned: listed for refine_kernel, which writes P and enters it in the arg-max; here it counts as 0
                const int64_t k = kh + (int64_t)(l0 + c8 + i) * UD_H;
                if (!(R2 < q.refine_r2) && k < p.Nf && refine_push(q.list, db, k)) { pf[i] = 0.f; continue; }
                if (!(R2 > 0.25f * Nt_f * Nt_f)) continue;
                const double XC = (double)xc[i], XS = (double)xs[i], Ad = 2.0 * (double)cc[i], Bd = 2.0 * (double)cs[i];
                const double R2d = Ad * Ad + Bd * Bd, x2 = XC * XC, y2 = XS * XS, Sd = x2 + y2;
                const double DRd = (x2 - y2) * Ad + 2.0 * XC * XS * Bd;
                double val;
                if (R2d < (1.0 - 1e-6) * (1.0 - 1e-6) * Nt * Nt) val = fmax(2.0 * (Sd * Nt - DRd), 0.0) / (Nt * Nt - R2d);
                else { const double R = sqrt(R2d); val = fmax(Sd + DRd / R, 0.0) / (Nt + R); }      // reading G7
                pf[i] = (float)(val * inv2var);
            }
        }
        #pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int64_t k = kh + (int64_t)(l0 + c8 + i) * UD_H;
            if (k < p.Nf) {
                if (q.P) q.P[db * q.p_stride + k] = pf[i];
                const u64 key = ((u64)__float_as_uint(fmaxf(pf[i], 0.f)) << 32) | (u64)(0xffffffffu - (unsigned)k);
                best = (key > best) ? key : best;
            }
        }
    }
    if (q.peak_idx == nullptr) return;
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) { const u64 other = __shfl_down_sync(0xffffffffu, best, o); best = (other > best) ? other : best; }
    if (lane == 0 && live) {                                            // step 7: order-free packed arg-max, lowest k on ties (reading G9)
        atomicMax(q.peak64 + db, best);
        __threadfence();
        const unsigned done = atomicAdd(q.counter + db, 1u);
        if (done == 4u * (unsigned)p.nfb - 1u) {                        // 4 warps per series per frequency block: the last one publishes
            __threadfence();
            const u64 fin = atomicMax(q.peak64 + db, 0ull);
            q.peak_idx[db] = (int32_t)(0xffffffffu - (unsigned)(fin & 0xffffffffull));
            q.peak_val[db] = __uint_as_float((unsigned)(fin >> 32));
        }
    }
}

// grid.x = ceil(B / 2) * nsplit * nfb (frequency block fastest), US_THREADS threads, UD_SMEM bytes, two CTAs per SM.
// FUSED_PRE (short series, as in accum_umma_small_kernel): steps 1-2 run here -- the 128 loader threads of each series form its mean
// and variance over the WHOLE series (fixed order: every CTA of the series gets the identical values) and the exact phases of the
// samples they stage, straight from t and x; no record arrays, no pre-pass launches.  The first CTA of a series publishes the
// variance partial and resets the arg-max cell (host: only where no other CTA of the series can reach its epilogue first).
// WEIGHTED (weighted generalised periodogram, never with FUSED_PRE): as in accum_umma_small_kernel.
template <bool FUSED_PRE, bool WEIGHTED = false>
__global__ void __launch_bounds__(US_THREADS, 2) accum_umma_duo_kernel(const UmmaDuoParams q)
{
    const UmmaParams& p = q.u;
    extern __shared__ __align__(128) unsigned char um_smem[];
    float4* rec_all = reinterpret_cast<float4*>(um_smem + UD_STAGES * UD_STAGE_BYTES);            // [series][2][UM_TS] {X/sigma, pA32, v32, w32}
    float* recw_all = reinterpret_cast<float*>(um_smem + UD_STAGES * UD_STAGE_BYTES + UD_REC_BYTES);   // [series][2][UM_TS] normalised weight (WEIGHTED)
    uint64_t* bars = reinterpret_cast<uint64_t*>(um_smem + UD_STAGES * UD_STAGE_BYTES + UD_REC_BYTES + UD_RECW_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * UD_STAGES + 2);

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t bp = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * UD_FPB;
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const int64_t n_samp = j_end - j_begin;
    const int nks = (int)((n_samp + UM_KS - 1) / UM_KS);
    const int flush_ksteps = max(1, p.flush_ksteps);

    const uint32_t s_stage = smem_u32(um_smem), s_bar = smem_u32(bars);
    const uint32_t bar_accf = s_bar + 8u * (2 * UD_STAGES), bar_acce = bar_accf + 8u;
#define UD_FULL(s) (s_bar + 8u * (unsigned)(s))
#define UD_EMPTY(s) (s_bar + 8u * (unsigned)(UD_STAGES + (s)))

    if (tid == 0) {
        for (int s = 0; s < UD_STAGES; ++s) { mbar_init(UD_FULL(s), US_GEN_WARPS); mbar_init(UD_EMPTY(s), 1); }
        mbar_init(bar_accf, 1);
        mbar_init(bar_acce, US_GEN_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == US_GEN_WARPS) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"((uint32_t)UD_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);

    if (w < US_GEN_WARPS) {
        // ===================== producers: steps 3 (operand tiles) and 5 (drain) =====================
        // Everything that does not change from k-step to k-step is formed once, here, and the loop below only advances a few
        // 32-bit counters: the loop overhead was 40 % of the instructions of this generation-bound kernel (round 2).
        // record loader role: thread tid -> series tid >> 7, sample tid & 127 of the tile
        const unsigned ls = tid >> 7, lj = tid & 127u;
        const int64_t lb = 2 * bp + ls;
        const bool l_live = lb < q.B;
        const float* recAx = &p.recA[(l_live ? lb : 0) * p.Nt + j_begin].x;      // .x of the split's first record (stride 4 floats)
        const ulonglong2* recB = p.recB + (l_live ? lb : 0) * p.Nt + j_begin;
        float xs;
        double mean = 0.0, t0 = 0.0;
        const double* tb = nullptr; const float* xb = nullptr;
        if (FUSED_PRE) {
            // steps 1-2: mean, then sum (x - mean)^2, of series `ls` by its 128 loader threads (warps 4 ls ... 4 ls + 3)
            tb = p.t + (l_live ? lb : 0) * p.t_stride; xb = p.x + (l_live ? lb : 0) * p.x_stride;
            double* red = reinterpret_cast<double*>(rec_all);                     // 8 doubles of scratch (the record tiles are not in use yet)
            double a0 = 0.0;
            for (int64_t j = lj; j < p.Nt; j += 128) a0 += (double)__ldg(xb + j);
            #pragma unroll
            for (int o = 16; o > 0; o >>= 1) a0 += __shfl_down_sync(0xffffffffu, a0, o);
            if (lane == 0) red[w] = a0;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            const double sum_x = ((red[4 * ls] + red[4 * ls + 1]) + red[4 * ls + 2]) + red[4 * ls + 3];      // fixed order
            mean = sum_x / (double)p.Nt;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            double a1 = 0.0;
            for (int64_t j = lj; j < p.Nt; j += 128) { const double d = (double)__ldg(xb + j) - mean; a1 += d * d; }
            #pragma unroll
            for (int o = 16; o > 0; o >>= 1) a1 += __shfl_down_sync(0xffffffffu, a1, o);
            if (lane == 0) red[w] = a1;
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            const double q2 = ((red[4 * ls] + red[4 * ls + 1]) + red[4 * ls + 2]) + red[4 * ls + 3];
            asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");   // `red` is the record tiles from here on
            if (lj == 0 && l_live && sp == 0 && fb == 0) { p.part_var_out[lb] = q2; p.part_sum_out[lb] = sum_x; p.peak64[lb] = 0ull; p.counter[lb] = 0u; }
            xs = l_live ? x_scale(&q2, 1, p.Nt) : 0.f;                            // steps 6-7 recompute exactly this from part_var_out
            t0 = __ldg(tb);                                                       // time origin (reading G6)
        } else {
            xs = l_live ? (p.unit_x ? 1.f : x_scale(p.part_var + lb * p.nparts, p.nparts, p.Nt)) : 0.f;
        }
        const int n_samp_i = (int)n_samp;                                         // split_len < 2^31
        float pre_x = 0.f, pre_w = 1.f; u64 pre_u = 0ull, pre_v = 0ull;
        bool pre_ok = false;
        const float* recWx = WEIGHTED ? &p.recW[(l_live ? lb : 0) * p.Nt + j_begin].x : nullptr;
        auto prefetch = [&](int jt) {                                             // this thread's record of a tile, relative to j_begin
            pre_ok = l_live && jt < n_samp_i;
            if (!pre_ok) return;
            if (FUSED_PRE) {
                const int64_t j = j_begin + jt;
                pre_x = (float)((double)__ldg(xb + j) - mean);                    // X_j rounded to fp32 once (G4)
                const double tp = __ldg(tb + j) - t0;
                pre_u = frac_fixed64(p.f_min, tp, nullptr);
                pre_v = frac_fixed64(p.df, tp, nullptr);
            } else { pre_x = __ldg(recAx + 4 * jt); const ulonglong2 r = __ldg(recB + jt); pre_u = r.x; pre_v = r.y; }
            if (WEIGHTED) pre_w = __ldg(recWx + 4 * jt);
        };
        prefetch((int)lj);
        float4* rec_mine = rec_all + (ls * 2) * UM_TS + lj;                       // this thread's slot of its series' tile, buffer 0
        float* recw_mine = recw_all + (ls * 2) * UM_TS + lj;
        // A task: row m = tid & 127 = (series m >> 6, fine value m & 63), 4 samples `chunk` of the k-step
        const unsigned m = tid & 127u, a_s = m >> 6, a_h = m & 63u;
        const int chunk = (int)(tid >> 7);
        const float4* rec_a = rec_all + (a_s * 2) * UM_TS + chunk * 4;            // + buffer * UM_TS + first sample of the k-step
        const float* recw_a = recw_all + (a_s * 2) * UM_TS + chunk * 4;
        const uint32_t a_dst = s_stage + (uint32_t)chunk * (UM_A_BYTES / 2) + m * 16u;
        // B task (128 per k-step: threads 0..127 on even k-steps, 128..255 on odd ones): series (tid >> 6) & 1, K chunk (tid >> 5) & 1, coarse value tid & 31
        const unsigned b_s = (tid >> 6) & 1u, bc = (tid >> 5) & 1u, b_l = tid & 31u, b_par = (tid >> 7) & 1u;
        const float4* rec_b = rec_all + (b_s * 2) * UM_TS + (int)bc * 4;
        const uint32_t b_dst = s_stage + 3 * UM_A_BYTES + bc * (UM_A_BYTES / 2) + (b_s * 64u + b_l) * 16u;
        // drain role: TMEM lane quadrant q4 (series q4 >> 1), Re (0) / Im (1) columns of that series' diagonal block
        const unsigned q4 = w & 3u, part = w >> 2, d_s = q4 >> 1;
        const int64_t db = 2 * bp + d_s;
        const bool d_live = db < q.B;
        float* ws_unit = p.ws + (((d_live ? db : 0) * p.nsplit + sp) * 4) * p.Nf;
        const int64_t k0 = kb + (int64_t)((32u * q4 + lane) & 63u);
        const uint32_t t_drain = tmem + ((32u * q4) << 16) + 64u * d_s + (uint32_t)UD_L * part;
        int flushes = 0;
        int s = 0;                                                              // ring stage of this k-step
        uint32_t ph_empty = 1u;                                                 // parity to wait for on EMPTY[s]
        int sb = 0, buf = 0;                                                    // first sample of the k-step within the tile; tile buffer
        int left = n_samp_i - chunk * 4;                                        // samples left from this thread's first A sample on
        int j_tile = (int)lj;                                                   // this thread's record of the tile being loaded, relative to j_begin

        for (int ks = 0; ks < nks; ) {
          const int ks_begin = ks;
          const int ks_end = min(nks, ks + flush_ksteps);                       // one drain window: the hot loop holds no drain code (registers)
          #pragma unroll 1
          for (; ks < ks_end; ++ks) {
            if (sb == 0) {                                                      // next record tile of both series
                float4 r = make_float4(0.f, 0.f, 0.f, 0.f);                     // pad: X = 0, phases 0
                if (pre_ok) {
                    const u64 pa = pre_u + (u64)kb * pre_v;                     // u + kb v (mod 1, 64-bit wrap; reading G3)
                    r.x = WEIGHTED ? pre_x * xs * pre_w : pre_x * xs;
                    r.y = __uint_as_float((unsigned)((pa + 0x80000000ull) >> 32));
                    r.z = __uint_as_float((unsigned)((pre_v + 0x80000000ull) >> 32));
                    r.w = __uint_as_float((unsigned)(((u64)UD_H * pre_v + 0x80000000ull) >> 32));
                }
                rec_mine[buf * UM_TS] = r;
                if (WEIGHTED) recw_mine[buf * UM_TS] = pre_ok ? pre_w * pre_w : 0.f;
                j_tile += UM_TS;                                                // prefetch this thread's record of the following tile
                prefetch(j_tile);
                asm volatile("bar.sync 1, %0;" :: "n"(US_GEN_WARPS * 32) : "memory");
            }
            const uint32_t st_off = (uint32_t)s * UD_STAGE_BYTES;
            mbar_wait(UD_EMPTY(s), ph_empty);                                   // the MMAs that read this stage have completed
            {
                const float4* ra = rec_a + buf * UM_TS + sb;
                const float* rw = recw_a + buf * UM_TS + sb;
#ifndef LSP_UD_DBG_NOA
                if (left >= 4) um_gen_a<false, WEIGHTED>(ra, 0, a_h, a_dst + st_off, 4, rw);  // `left` is warp-uniform
                else um_gen_a<true, WEIGHTED>(ra, 0, a_h, a_dst + st_off, max(0, left), rw);
#else
                (void)ra; (void)rw;
#endif
            }
#ifndef LSP_UD_DBG_NOB
            if (((unsigned)ks & 1u) == b_par) ud_gen_b(rec_b + buf * UM_TS + sb, 0, b_l, b_dst + st_off);
#endif
#ifndef LSP_UD_DBG_NOFENCE
            fence_proxy_async();                                                // generic-proxy stores -> visible to the tensor core
#endif
            __syncwarp();
            if (lane == 0) mbar_arrive(UD_FULL(s));
            left -= UM_KS;
            sb += UM_KS;
            if (sb == UM_TS) { sb = 0; buf ^= 1; }
            if (++s == UD_STAGES) { s = 0; ph_empty ^= 1u; }
          }
            const bool last = (ks == nks);
            {
                mbar_wait(bar_accf, (uint32_t)flushes & 1u);                    // every MMA issued so far has completed
                tc_fence_after();
                if (q.fuse) {                                                   // (host guarantees: this is the only drain of the CTA)
                    ud_finish16(q, tmem + ((32u * q4) << 16) + 64u * d_s + 16u * part, db, d_live, k0, 16u * part, lane);   // (one short window of noise-like sums: no compensation, it costs 5 % here)
                } else {
                const float nk = (float)(ks - ks_begin);                // k-steps of this window
                ud_drain(t_drain, ws_unit + (int64_t)part * p.Nf, k0, p.Nf, flushes == 0, d_live, p.trunc_ulps < 0.f ? nk : 0.f,
                         0.6366198f / (16.f * nk * (p.unit_x ? TC_MEAN_ABS_COS : TC_MEAN_ABS_PRODUCT)));
                ud_drain(t_drain + 128u, ws_unit + (int64_t)(2 + part) * p.Nf, k0, p.Nf, flushes == 0, d_live);   // D_V with D_W (see lsp_accum_umma_small.cuh)
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_acce);
                ++flushes;
            }
        }
    } else if (lane == 0) {
        // ===================== step 4: the single MMA-issuing thread =====================
        int kin = 0, flushes = 0;
        for (int ks = 0; ks < nks; ++ks) {
            const int s = ks & (UD_STAGES - 1);
            const uint32_t ph = (uint32_t)(ks / UD_STAGES) & 1u;
            mbar_wait(UD_FULL(s), ph);
            tc_fence_after();
            const uint32_t a0 = s_stage + (uint32_t)s * UD_STAGE_BYTES, b0 = a0 + 3 * UM_A_BYTES;
            const uint64_t dAh = umma_desc(a0, UM_A_BYTES / 2, 128), dAl = umma_desc(a0 + UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dAv = umma_desc(a0 + 2 * UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dBh = umma_desc(b0, UM_A_BYTES / 2, 128), dBl = umma_desc(b0 + UM_A_BYTES, UM_A_BYTES / 2, 128);
            const uint64_t dBv = umma_desc(b0 + 2 * UM_A_BYTES, UM_A_BYTES / 2, 128);
#ifndef LSP_UD_DBG_NOMMA
            tc_mma_f16(tmem, dAh, dBh, UD_IDESC, kin > 0 ? 1u : 0u);
            tc_mma_f16(tmem, dAl, dBh, UD_IDESC, 1u);
            tc_mma_f16(tmem, dAh, dBl, UD_IDESC, 1u);
            tc_mma_f16(tmem + 128u, dAv, dBv, UD_IDESC, kin > 0 ? 1u : 0u);
#else
            (void)dAh; (void)dAl; (void)dAv; (void)dBh; (void)dBl; (void)dBv;
#endif
            tc_commit(UD_EMPTY(s));
            const bool last = (ks == nks - 1);
            if (++kin == flush_ksteps || last) {
                tc_commit(bar_accf);
                if (!last) { mbar_wait(bar_acce, (uint32_t)flushes & 1u); tc_fence_after(); }
                ++flushes; kin = 0;
            }
        }
    }
#undef UD_FULL
#undef UD_EMPTY

    tc_fence_before();
    __syncthreads();
    if (w == US_GEN_WARPS) {
        __syncwarp();
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((uint32_t)UD_TMEM_COLS) : "memory");
    }
}

}  // namespace lsp
