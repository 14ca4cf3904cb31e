// lsp_plan.h -- host-only launch planner (no CUDA calls): picks the accumulate kernel variant
// (K adjacent frequencies per thread, T threads per CTA) and the number of time-axis splits.
//
// The accumulate grid is B * nfb * nsplit equal-sized CTAs ("units") handed out by the hardware
// block scheduler.  Three effects decide the run time and are modelled here (constants measured on
// B200):
//   fill      frequencies actually needed / frequencies the nfb blocks cover (ragged last block)
//   body      FFMA2 stream vs per-sample anchor overhead: 6K / (6K + 16) FMA-pipe cycles
//   waves     units / CTA slots is rarely an integer; the last, partly filled wave costs a full
//             unit time (measured: 8.28 waves ran as 9 => 8 % idle), so nsplit is chosen to make
//             the wave count large and just below an integer
// plus a fixed per-unit cost (outer-sum init, workspace write) that penalises very short splits.
#pragma once
#include <cstdint>

namespace lsp {

constexpr int PLAN_REC_ROTATION = 1, PLAN_REC_THREE_TERM = 2, PLAN_REC_THREE_TERM_Z = 3, PLAN_REC_MMA = 4, PLAN_REC_UMMA = 5;
constexpr int PLAN_UMMA_TS = 128;                                  // samples per record tile (lsp_accum_umma.cuh)
constexpr int PLAN_MMA_FPB = 8192, PLAN_MMA_TS = 128;              // frequencies per CTA, samples per tile (lsp_accum_mma.cuh)
constexpr int PLAN_TILE_PAIR = 512, PLAN_TILE_Z = 256;

struct PlanChoice {
    int K = 0, T = 0, nsplit = 1, rec = 0, nfb = 0, ctas_per_sm = 0;
    int L = 0;                      // tcgen05 form: coarse extent (frequencies per CTA = 128 L); 0 otherwise
    int64_t split_len = 0;
    double score = 0.0;
};

struct PlanOverrides { int64_t K = 0, T = 0, nsplit = 0, rec = 0, L = 0; };

inline bool plan_valid_K(int rec, int K) {
    if (K < 4 || K > 32 || (K % 4) != 0) return false;
    return rec == PLAN_REC_THREE_TERM_Z ? true : K <= 24;
}

inline int plan_max_threads(int rec, int K) { return (rec == PLAN_REC_THREE_TERM_Z && K >= 28) ? 128 : 256; }

// registers per thread as compiled (ptxas -v, kept in step with build_ptxas.log by tests/test_gpu_plan.py)
inline int plan_regs(int rec, int K) {
    static const int z[9]    = {0, 64, 96, 126, 128, 158, 128, 168, 168};      // K = 4..32
    static const int pair[7] = {0, 80, 128, 128, 184, 248, 255};               // K = 4..24
    return rec == PLAN_REC_THREE_TERM_Z ? z[K / 4] : pair[K / 4];
}

inline int64_t plan_smem_bytes(int rec, int K, int T) {
    if (rec == PLAN_REC_THREE_TERM_Z) return (int64_t)PLAN_TILE_Z * 24 + (int64_t)T * (4 * K + 1) * 4;
    return (int64_t)3 * (PLAN_TILE_PAIR / 2) * 16 + (int64_t)16 * K * T;
}

// resident CTAs per SM (B200: 64K registers, 228 KB shared memory with 1 KB reserved per CTA, 64 warps)
inline int plan_ctas_per_sm(int rec, int K, int T) {
    const int regs = (plan_regs(rec, K) + 7) / 8 * 8;
    int by_regs = 65536 / (regs * T);
    int by_smem = (int)((int64_t)233472 / (plan_smem_bytes(rec, K, T) + 1024));
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

// tcgen05 form, cost model (SM cycles at the nominal clock, measured on B200): cycles one SM spends per k-step of
// 8 samples of ONE CTA's 128 L frequencies.  L = 128 is bound by the tensor pipe (4 MMAs m128n256k16 = 512 cycles at
// the nominal clock; the measured figure includes the power-capped clock of long runs and is higher without the
// coarse-operand table); L <= 64 by the generation of the fine operand A (lsp_accum_umma_small.cuh), two CTAs per SM:
// measured 458 / 566 / 698 SM cycles per CTA k-step for L = 16 (three CTAs per SM) / 32 / 64 (C3 and C4, profiles/r01_bench_auto.md).
inline double plan_umma_kstep_cycles(int L, int nfb) {
    switch (L) {
        case 16: return 458.0;
        case 32: return 566.0;
        case 64: return 698.0;
        default: return nfb >= 3 ? 950.0 : 1150.0;
    }
}
inline int plan_umma_ctas_per_sm(int L) { return L >= 128 ? 1 : (L == 16 ? 3 : 2); }
inline double plan_umma_fixed_cycles(int L) { return (L >= 128 ? 8000.0 : 9000.0) + 93.0 * L; }   // per CTA: set-up + final drain (2 KB L at ~22 B per cycle per SM)

inline double plan_umma_cycles(int sm_count, int64_t units, int64_t split_len, int L, int nfb) {
    const int cps = plan_umma_ctas_per_sm(L);
    const int64_t slots = (int64_t)cps * sm_count;
    const int64_t waves = (units + slots - 1) / slots;
    const double share = units >= slots ? (double)cps : (double)((units + sm_count - 1) / sm_count);   // CTAs sharing an SM
    return (double)waves * ((double)((split_len + 7) / 8) * plan_umma_kstep_cycles(L, nfb) * share + plan_umma_fixed_cycles(L));
}

// Tensor-core forms: a CTA owns `fpb` frequencies (8,192 mma.sync; 128 L tcgen05, L = 16 / 32 / 64 / 128); the time
// split and (tcgen05) L are free.  Picks the (L, nsplit) with the fewest estimated cycles.
inline PlanChoice plan_choose_mma(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov, int rec = PLAN_REC_MMA)
{
    PlanChoice best;
    double best_cycles = 0.0;
    const int Ls[4] = {128, 64, 32, 16};
    for (int li = 0; li < (rec == PLAN_REC_UMMA ? 4 : 1); ++li) {
        const int L = rec == PLAN_REC_UMMA ? Ls[li] : 0;
        if (rec == PLAN_REC_UMMA && ov.L && ov.L != L) continue;
        const int FPB = rec == PLAN_REC_UMMA ? 128 * L : PLAN_MMA_FPB, TS = rec == PLAN_REC_UMMA ? PLAN_UMMA_TS : PLAN_MMA_TS;
        const int cps = rec == PLAN_REC_UMMA ? plan_umma_ctas_per_sm(L) : 1;
        const int64_t nfb = (Nf + FPB - 1) / FPB;
        const int64_t max_splits = (Nt + TS - 1) / TS;
        int64_t cap = ((int64_t)1 << 31) / (B * 16 * Nf);
        if (cap < 1) cap = 1;
        int64_t hi = max_splits < cap ? max_splits : cap;
        if (hi > 1024) hi = 1024;
        int64_t lo = 1;
        if (ov.nsplit) { lo = hi = (ov.nsplit < max_splits ? ov.nsplit : max_splits); }
        PlanChoice cand;                                            // best time split for this L
        double cand_cycles = 0.0;
        for (int64_t n = lo; n <= hi; ++n) {
            int64_t len = (Nt + n - 1) / n;
            len = (len + TS - 1) / TS * TS;
            const int64_t n_eff = (Nt + len - 1) / len;
            if (n_eff != n && !ov.nsplit) continue;
            const int64_t units = B * nfb * n_eff;
            double cycles;
            if (rec == PLAN_REC_UMMA) cycles = plan_umma_cycles(sm_count, units, len < Nt ? len : Nt, L, (int)nfb);
            else cycles = (double)((units + sm_count - 1) / sm_count) * ((double)len + 300.0);
            if (cand.K == 0 || cycles < cand_cycles * 0.9975) {     // near-ties: fewer splits
                cand.K = rec == PLAN_REC_UMMA ? L : 32; cand.L = L;
                cand.T = rec == PLAN_REC_UMMA ? (L >= 128 ? 544 : 288) : 256;
                cand.nsplit = (int)n_eff; cand.rec = rec; cand.nfb = (int)nfb;
                cand.ctas_per_sm = cps; cand.split_len = len; cand_cycles = cycles;
                cand.score = (double)Nf / (double)(nfb * FPB);
            }
        }
        if (cand.K && (best.K == 0 || cand_cycles < best_cycles * 0.97)) { best = cand; best_cycles = cand_cycles; }   // near-ties: the wider tile
    }
    return best;
}

// FP32-pipe forms (rec 1-3): K adjacent frequencies per thread, T threads per CTA, nsplit time splits.
inline PlanChoice plan_choose_fp32(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov, int rec)
{
    const int tile = rec == PLAN_REC_THREE_TERM_Z ? PLAN_TILE_Z : PLAN_TILE_PAIR;
    const int64_t max_splits_tile = (Nt + tile - 1) / tile;
    int Ts[3] = {128, 64, 32};                                      // automatic candidates (256 only on request)
    int nT = 3;
    if (ov.T) { Ts[0] = (int)ov.T; nT = 1; }
    PlanChoice best;
    for (int K = 32; K >= 4; K -= 4) {
        if (!plan_valid_K(rec, K)) continue;
        if (ov.K && ov.K != K) continue;
        for (int ti = 0; ti < nT; ++ti) {
            const int T = Ts[ti];
            if (T > plan_max_threads(rec, K)) continue;
            const int cta = plan_ctas_per_sm(rec, K, T);
            if (cta < 1) continue;
            const int64_t fb = (int64_t)K * T;
            const int64_t nfb = (Nf + fb - 1) / fb;
            const double fill = (double)Nf / (double)(nfb * fb);
            const double body = 6.0 * K / (6.0 * K + 16.0);
            const double wps = cta * T / 128.0;                     // warps per SM sub-partition
            const double occ = wps >= 3.0 ? 1.0 : (wps >= 2.0 ? 0.93 : (wps >= 1.0 ? 0.72 : 0.72 * wps));
            const int64_t slots = (int64_t)cta * sm_count;
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
                const int64_t units = B * nfb * n_eff;
                const double wave = plan_wave_eff(units, slots);
                const double avg_len = (double)Nt / (double)n_eff;
                const double unit = avg_len / (avg_len + 40.0);
                const double score = fill * body * occ * wave * unit;
                if (score > best.score * 1.0025 || best.K == 0) {   // prefer earlier (larger K, fewer splits) on near-ties
                    best.K = K; best.T = T; best.nsplit = (int)n_eff; best.rec = rec; best.nfb = (int)nfb;
                    best.ctas_per_sm = cta; best.split_len = len; best.score = score;
                }
            }
        }
    }
    return best;
}

// Estimated run time in SM cycles at the nominal clock (for choosing between the forms; constants measured on B200):
//   FP32 z form: 6 lane-ops per term on 128 lanes per SM at the modelled efficiency `score`;
//   tcgen05 form: ~950 cycle-equivalents per k-step of 8 samples x 16,384 frequencies (power-capped clocks
//   included; 1,150 without the coarse-operand table) plus ~20,000 per CTA (set-up, final drain), per wave.
inline double plan_est_cycles(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanChoice& pc)
{
    if (pc.rec == PLAN_REC_UMMA)
        return plan_umma_cycles(sm_count, B * (int64_t)pc.nfb * pc.nsplit, pc.split_len, pc.L, pc.nfb);
    const double lane_ops = pc.rec == PLAN_REC_ROTATION ? 8.0 : 6.0;
    return (double)B * (double)Nt * (double)Nf * lane_ops / (128.0 * sm_count * (pc.score > 1e-6 ? pc.score : 1e-6)) + 4000.0;
}

constexpr int64_t PLAN_TC_MIN_NT = 512;   // tensor-core forms: V takes one fp16 pass, |dP|/P ~ 4e-4 / sqrt(Nt)

// rec = 0 (automatic): the tcgen05 form when it is accurate (Nt >= 512) and the model says it is faster,
// else the FP32 z form.  An explicit rec is always honoured.
inline PlanChoice plan_choose(int sm_count, int64_t B, int64_t Nt, int64_t Nf, const PlanOverrides& ov)
{
    if (ov.rec == PLAN_REC_MMA || ov.rec == PLAN_REC_UMMA) return plan_choose_mma(sm_count, B, Nt, Nf, ov, (int)ov.rec);
    if (ov.rec) return plan_choose_fp32(sm_count, B, Nt, Nf, ov, (int)ov.rec);
    const PlanChoice z = plan_choose_fp32(sm_count, B, Nt, Nf, ov, PLAN_REC_THREE_TERM_Z);
    if (Nt < PLAN_TC_MIN_NT || ov.K || ov.T) return z;               // K / T overrides address the FP32 kernels
    const PlanChoice u = plan_choose_mma(sm_count, B, Nt, Nf, ov, PLAN_REC_UMMA);
    return plan_est_cycles(sm_count, B, Nt, Nf, u) < plan_est_cycles(sm_count, B, Nt, Nf, z) ? u : z;
}

}  // namespace lsp
