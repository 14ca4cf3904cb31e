// lsp_plan.h -- host-only launch planner (no CUDA calls): picks the form of steps 3-5 (FP32 pipe or tensor cores),
// its tile (K adjacent frequencies per thread and T threads per CTA; or the coarse extent L of a tcgen05 tile), the
// number of time-axis splits and, for the table-fed CTA-pair form, the time chunks that bound the table.
//
// The accumulate grid is B * nfb * nsplit equal-sized CTAs ("units") handed out by the hardware block scheduler.
// The run time of the FP32 form is modelled as waves x (time of one wave of resident CTAs), score = ideal cycles / estimate
// (constants measured on B200).  What enters:
//   fill      frequencies actually needed / frequencies the nfb blocks cover (ragged last block): through the CTA count
//   body      FFMA2 stream vs the per-sample fixed cost (anchor, loop, register moves): 6K / (6K + 44) FMA-pipe cycles per
//             sample and warp (measured on B200 for K = 16 ... 48: 232 cycles at K = 32, 144 at K = 16; round 2)
//   waves     units / CTA slots is rarely an integer; the last, partly filled wave costs a full
//             unit time (measured: 8.28 waves ran as 9 => 8 % idle), so nsplit is chosen to make
//             the wave count large and just below an integer
// plus a fixed per-unit cost (outer-sum init, workspace write) that penalises very short splits.
#pragma once
#include <cstdint>

namespace lsp {

constexpr int PLAN_PIPE_FP32 = 1, PLAN_PIPE_TENSOR = 2;            // = LSP_PIPE_* of include/lsp.h
constexpr int PLAN_UMMA_TS = 128;                                  // samples per record tile of the tcgen05 kernels
constexpr int PLAN_UMMA_TS_SMALL = 32;                             // granularity of the time splits of the short-grid tcgen05 forms
constexpr int PLAN_TILE_Z = 256;                                   // samples per tile of the FP32-pipe kernel
constexpr int64_t PLAN_TABLE_BYTES_PER_SAMPLE = 3072;              // CTA-pair form: fine-operand table (lsp_accum_umma_pair2.cuh)
constexpr int64_t PLAN_TABLE_BUDGET_DEFAULT = (int64_t)1 << 30;    // bytes of workspace the table may take: longer series run in time chunks
constexpr int64_t PLAN_TABLE_MIN_CHUNK = 2048;                     // a chunk shorter than this (batches of many long series) rules the pair form out

struct PlanChoice {
    int K = 0, T = 0, nsplit = 1, pipe = 0, nfb = 0, ctas_per_sm = 0;
    int L = 0;                      // tcgen05 forms: coarse extent (frequencies per CTA = 128 L); 0 otherwise
    int nchunks = 1;                // CTA-pair form (L = 128): time chunks, each with its own table pre-pass + accumulate launch
    int64_t chunk_len = 0;          //   samples per chunk (multiple of 128; the last chunk may be shorter); 0 otherwise
    int64_t split_len = 0;
    double score = 0.0;
};

struct PlanOverrides { int64_t K = 0, T = 0, nsplit = 0, pipe = 0, L = 0, table_budget = 0, table_series = 1; int max_K = 32; /* FP32 form: widest thread tile considered */ };

inline bool plan_valid_K(int K) { return K >= 4 && K <= 32 && (K % 4) == 0; }

inline int plan_max_threads(int K) { return K >= 28 ? 128 : 256; }

// registers per thread of accum_z_kernel<K> as compiled (ptxas -v; tests/test_plan.py checks this table against build_ptxas.log)
inline int plan_regs(int K) {
    static const int z[9] = {0, 64, 96, 122, 128, 154, 128, 168, 168};         // K = 4..32
    return z[K / 4];
}

constexpr int64_t PLAN_FOLD_SAMPLES = 2048;                        // default fold interval of the FP32-pipe kernel's register partials
// a split inside one fold interval needs no shared-memory accumulators (accum_z_kernel<..., DIRECT>)
inline int64_t plan_smem_bytes(int K, int T, bool direct = false) { return (int64_t)PLAN_TILE_Z * 24 + (direct ? 0 : (int64_t)T * (4 * K + 1) * 4); }

// resident CTAs per SM (B200: 64K registers, 228 KB shared memory with 1 KB reserved per CTA, 64 warps)
inline int plan_ctas_per_sm(int K, int T, bool direct = false) {
    const int regs = (plan_regs(K) + 7) / 8 * 8;
    int by_regs = 65536 / (regs * T);
    int by_smem = (int)((int64_t)233472 / (plan_smem_bytes(K, T, direct) + 1024));
    int by_warps = 2048 / T;
    int c = by_regs < by_smem ? by_regs : by_smem;
    if (by_warps < c) c = by_warps;
    if (c > 32) c = 32;
    return c;
}

inline double plan_wave_eff(int64_t units, int64_t slots) {
    if (units <= slots) return (double)units / (double)slots;
    const int64_t waves = (units + slots - 1) / slots;
    return (double)units / (double)(waves * slots);
}

// tcgen05 forms, cost model (SM cycles at the nominal clock, measured on B200): cycles one SM spends per k-step of
// 8 samples of ONE CTA's 128 L frequencies.  L = 128 (CTA-pair form) is bound by the tensor pipe (3 MMA slots of
// m256n256 per pair and k-step; the figure includes the power-capped clock of long runs); L <= 64 by the generation
// of the fine operand A (lsp_accum_umma_small.cuh), two CTAs per SM: measured 458 / 566 / 698 SM cycles per CTA k-step
// for L = 16 (three CTAs per SM) / 32 / 64 (C3 and C4, profiles/r01_bench_auto.md).
inline double plan_umma_kstep_cycles(int L) {
    switch (L) {
        case 16: return 458.0;
        case 32: return 566.0;
        case 64: return 698.0;
        default: return 950.0;
    }
}
inline int plan_umma_ctas_per_sm(int L) { return L >= 128 ? 1 : (L == 16 ? 3 : 2); }
inline double plan_umma_fixed_cycles(int L) { return (L >= 128 ? 8000.0 : 9000.0) + 93.0 * L; }   // per CTA: set-up + final drain (2 KB L at ~22 B per cycle per SM)

inline double plan_umma_cycles(int sm_count, int64_t units, int64_t split_len, int L) {
    const int cps = plan_umma_ctas_per_sm(L);
    const int64_t slots = (int64_t)cps * sm_count;
    const int64_t waves = (units + slots - 1) / slots;
    const double share = units >= slots ? (double)cps : (double)((units + sm_count - 1) / sm_count);   // CTAs sharing an SM
    return (double)waves * ((double)((split_len + 7) / 8) * plan_umma_kstep_cycles(L) * share + plan_umma_fixed_cycles(L));
}
// table pre-pass of the CTA-pair form: 3 KB written per sample at the HBM write rate, ~1.1 device cycles per sample
// (measured: 0.55 ms at Nt = 1e6), plus a launch per chunk
inline double plan_table_cycles(int64_t samples, int nchunks) { return 1.1 * (double)samples + 8000.0 * nchunks; }

// Tensor-core forms: a CTA owns 128 L frequencies, L = 16 / 32 / 64 (both operands generated) or 128 (CTA pairs of
// 32,768 frequencies, table-fed; nfb is then even); the time split and L are free.  Picks the (L, nsplit) with the fewest estimated cycles.
inline PlanChoice plan_choose_tensor(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov, double* cycles_out = nullptr)
{
    PlanChoice best;
    double best_cycles = 0.0;
    const int Ls[4] = {128, 64, 32, 16};
    const int64_t budget = ov.table_budget > 0 ? ov.table_budget : PLAN_TABLE_BUDGET_DEFAULT;
    for (int li = 0; li < 4; ++li) {
        const int L = Ls[li];
        if (ov.L && ov.L != L) continue;
        // granularity of the time splits: the record tile (128 samples) for the table-fed pair form; 32 samples (4 k-steps) for the
        // forms that generate both operands, so that short series (C1, C2) can be cut into many short CTAs: there the length of
        // ONE CTA's k-step chain is what a call costs
        const int FPB = 128 * L, TS = L >= 128 ? PLAN_UMMA_TS : PLAN_UMMA_TS_SMALL;
        const int cps = plan_umma_ctas_per_sm(L);
        int64_t nfb = (Nf + FPB - 1) / FPB;
        int nchunks = 1;
        int64_t chunk_len = Nt;
        if (L == 128) {
            nfb = (nfb + 1) & ~(int64_t)1;                          // CTA pairs
            int64_t max_chunk = budget / (PLAN_TABLE_BYTES_PER_SAMPLE * (ov.table_series > 0 ? ov.table_series : 1)) / TS * TS;
            if (max_chunk < (Nt < PLAN_TABLE_MIN_CHUNK ? Nt : PLAN_TABLE_MIN_CHUNK)) {
                if (!ov.L) continue;                                // the table of this batch does not fit: narrower tiles
                if (max_chunk < TS) max_chunk = TS;                 // forced: honour it with the smallest chunks
            }
            if (Nt > max_chunk) {
                nchunks = (int)((Nt + max_chunk - 1) / max_chunk);
                chunk_len = ((Nt + nchunks - 1) / nchunks + TS - 1) / TS * TS;
                nchunks = (int)((Nt + chunk_len - 1) / chunk_len);
            }
        }
        const int64_t max_splits = (chunk_len + TS - 1) / TS;
        int64_t cap = ((int64_t)1 << 31) / (B * 16 * Nf);
        if (cap < 1) cap = 1;
        int64_t hi = max_splits < cap ? max_splits : cap;
        if (hi > 1024) hi = 1024;
        int64_t lo = 1;
        if (ov.nsplit) { lo = hi = (ov.nsplit < max_splits ? ov.nsplit : max_splits); }
        PlanChoice cand;                                            // best time split for this L
        double cand_cycles = 0.0;
        for (int64_t n = lo; n <= hi; ++n) {
            int64_t len = (chunk_len + n - 1) / n;
            len = (len + TS - 1) / TS * TS;
            const int64_t n_eff = (chunk_len + len - 1) / len;
            if (n_eff != n && !ov.nsplit) continue;
            const int64_t units = B * nfb * n_eff;
            double cycles = (double)nchunks * plan_umma_cycles(sm_count, units, len < chunk_len ? len : chunk_len, L);
            if (L == 128) cycles += plan_table_cycles(Nt * (ov.table_series > 0 ? ov.table_series : 1), nchunks);
            if (cand.K == 0 || cycles < cand_cycles * 0.9975) {     // near-ties: fewer splits
                cand.K = L; cand.L = L;
                cand.T = L >= 128 ? 544 : 288;
                cand.nsplit = (int)n_eff; cand.pipe = PLAN_PIPE_TENSOR; cand.nfb = (int)nfb;
                cand.ctas_per_sm = cps; cand.split_len = len; cand_cycles = cycles;
                cand.nchunks = nchunks; cand.chunk_len = L == 128 ? chunk_len : 0;
                cand.score = (double)Nf / (double)(nfb * FPB);
            }
        }
        if (cand.K && (best.K == 0 || cand_cycles < best_cycles * 0.97)) { best = cand; best_cycles = cand_cycles; }   // near-ties: the wider tile
    }
    if (cycles_out) *cycles_out = best_cycles;
    return best;
}

// FP32-pipe form: K adjacent frequencies per thread, T threads per CTA, nsplit time splits.
inline PlanChoice plan_choose_fp32(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov)
{
    const int tile = PLAN_TILE_Z;
    const int64_t max_splits_tile = (Nt + tile - 1) / tile;
    int Ts[3] = {128, 64, 32};                                      // automatic candidates (256 only on request)
    int nT = 3;
    if (ov.T) { Ts[0] = (int)ov.T; nT = 1; }
    PlanChoice best;
    for (int K = 32; K >= 4; K -= 4) {
        if (ov.K && ov.K != K) continue;
        if (!ov.K && K > ov.max_K) continue;
        for (int ti = 0; ti < nT; ++ti) {
            const int T = Ts[ti];
            if (T > plan_max_threads(K)) continue;
            if (plan_ctas_per_sm(K, T) < 1) continue;
            const int64_t fb = (int64_t)K * T;
            const int64_t nfb = (Nf + fb - 1) / fb;
            const double fill = (double)Nf / (double)(nfb * fb);
            const double body = 6.0 * K / (6.0 * K + 44.0);
            // workspace cap: B * nsplit * 16 bytes * Nf <= 2 GiB
            int64_t cap = ((int64_t)1 << 31) / (B * 16 * Nf);
            if (cap < 1) cap = 1;
            int64_t hi = max_splits_tile < cap ? max_splits_tile : cap;
            if (hi > 1024) hi = 1024;
            int64_t lo = 1;
            if (ov.nsplit) { lo = hi = (ov.nsplit < max_splits_tile ? ov.nsplit : max_splits_tile); }
            for (int64_t n = lo; n <= hi; ++n) {
                int64_t len = (Nt + n - 1) / n;
                len = (len + tile - 1) / tile * tile;
                const int64_t n_eff = (Nt + len - 1) / len;         // splits actually produced
                if (n_eff != n && !ov.nsplit) continue;             // duplicate of a smaller n
                const int cta = plan_ctas_per_sm(K, T, len <= PLAN_FOLD_SAMPLES);   // short splits keep their sums in registers: more CTAs per SM
                const int64_t slots = (int64_t)cta * sm_count;
                const int64_t units = B * nfb * n_eff;
                // CTAs actually resident per SM: `cta` when the grid fills the machine, fewer when it does not (C1, C2) -- then what
                // counts is how long ONE CTA takes, so short splits and small K win, not the per-term efficiency of a full machine
                const int64_t resident = units >= slots ? cta : (units + sm_count - 1) / sm_count;
                double wps = resident * T / 128.0;                  // warps per SM sub-partition
                if (wps < 1.0) wps = 1.0;
                const double occ = wps >= 3.0 ? 1.0 : (wps >= 2.0 ? 0.93 : 0.72);
                const int64_t waves = units >= slots ? (units + slots - 1) / slots : 1;
                const double avg_len = (double)Nt / (double)n_eff;
                const double est = (double)waves * (avg_len + 40.0) * (6.0 * K + 44.0) * wps / occ;   // SM cycles
                const double ideal = (double)B * (double)Nt * (double)Nf * 6.0 / (128.0 * sm_count);
                const double score = ideal / est;
                (void)fill; (void)body;
                if (score > best.score * 1.0025 || best.K == 0) {   // prefer earlier (larger K, fewer splits) on near-ties
                    best.K = K; best.T = T; best.nsplit = (int)n_eff; best.pipe = PLAN_PIPE_FP32; best.nfb = (int)nfb;
                    best.ctas_per_sm = cta; best.split_len = len; best.score = score;
                }
            }
        }
    }
    return best;
}

// Estimated run time in SM cycles at the nominal clock (for choosing between the forms; constants measured on B200):
//   FP32 form: 6 lane-ops per term on 128 lanes per SM at the modelled efficiency `score`;
//   tcgen05 forms: plan_umma_cycles per chunk (+ the table pre-pass of the CTA-pair form).
inline double plan_est_cycles(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanChoice& pc, int64_t table_series = 1)
{
    if (pc.pipe == PLAN_PIPE_TENSOR) {
        const int64_t len = pc.chunk_len ? pc.chunk_len : Nt;
        double c = (double)pc.nchunks * plan_umma_cycles(sm_count, B * (int64_t)pc.nfb * pc.nsplit, pc.split_len < len ? pc.split_len : len, pc.L);
        if (pc.L == 128) c += plan_table_cycles(Nt * table_series, pc.nchunks);
        return c;
    }
    return (double)B * (double)Nt * (double)Nf * 6.0 / (128.0 * sm_count * (pc.score > 1e-6 ? pc.score : 1e-6)) + 4000.0;
}

constexpr int64_t PLAN_TC_MIN_NT = 512;   // tensor-core forms: V takes one fp16 pass, |dP|/P ~ 4e-4 / sqrt(Nt)

// pipe = 0 (automatic): a tcgen05 form when it is accurate (Nt >= 512) and the model says it is faster,
// else the FP32 form.  An explicit pipe is always honoured.
inline PlanChoice plan_choose(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov)
{
    if (ov.pipe == PLAN_PIPE_TENSOR) return plan_choose_tensor(sm_count, B, Nt, Nf, ov);
    const PlanChoice z = plan_choose_fp32(sm_count, B, Nt, Nf, ov);
    if (ov.pipe == PLAN_PIPE_FP32 || Nt < PLAN_TC_MIN_NT || ov.K || ov.T) return z;   // K / T overrides address the FP32 kernel
    const PlanChoice u = plan_choose_tensor(sm_count, B, Nt, Nf, ov);
    if (u.K == 0) return z;
    return plan_est_cycles(sm_count, B, Nt, Nf, u, ov.table_series) < plan_est_cycles(sm_count, B, Nt, Nf, z) ? u : z;
}

}  // namespace lsp
