// lsp.cu -- host side of the C ABI declared in include/lsp.h: argument checks, launch plan,
// workspace, and the four enqueues (moments -> records -> accumulate -> finish).
// No CPU arithmetic on the data path: every step of SURVEY.md section 8(a) runs in a kernel.
#include "../../include/lsp.h"
#include "lsp_common.cuh"
#include "lsp_prepass.cuh"
#include "lsp_accum.cuh"
#include "lsp_accum_z.cuh"
#include "lsp_accum_mma.cuh"
#include "lsp_accum_umma.cuh"
#include "lsp_accum_umma_tab.cuh"
#include "lsp_accum_umma_pair.cuh"
#include "lsp_accum_umma_pair2.cuh"
#include "lsp_accum_umma_small.cuh"
#include "lsp_shared_gemm.cuh"
#include "lsp_accum_umma_duo.cuh"
#include "lsp_finish.cuh"
#include "lsp_fap.cuh"
#include "lsp_plan.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <new>

using namespace lsp;

namespace {

struct Plan {
    int K = 0, T = 0, nsplit = 0, rec = 0, nfb = 0, flush_tiles = 0, nparts = 0, launches = 0, L = 0;
    int mma_slots = 4;          // tensor-core forms: fp16-rate MMA slots issued per k-step of 8 samples (4 = hi+lo in fp16, 3 = 8-bit correction)
    int64_t split_len = 0, part_chunk = 0;
    const char* kernel_name = "";
};

}  // namespace

constexpr int TIMING_RING = 64;

struct lsp_ctx {
    int device = 0;
    int sm_count = 148;
    int last_cuda = 0;
    // tunables (0 = automatic)
    int64_t opt_K = 0, opt_T = 0, opt_nsplit = 0, opt_rec = 0, opt_flush = 0, opt_timing = 0, opt_btable = 0, opt_coarse = 0, opt_corr = 0, opt_pair = 0, opt_shared = 0, opt_duo = 0;
    cudaEvent_t ev[TIMING_RING][5] = {};                  // ring of per-call event sets (LSP_PARAM_TIMING)
    uint64_t timed_calls = 0;
    // workspace
    void* buf = nullptr;
    size_t buf_bytes = 0;
    // staging for the host-pointer entry points
    void* stage = nullptr;
    size_t stage_bytes = 0;
    Plan plan;
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int cuda_fail(lsp_ctx* h, cudaError_t e) {
    if (h) h->last_cuda = (int)e;
    return LSP_ECUDA;
}

#define LSP_CUDA(h, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((h), e_); } while (0)

struct DeviceGuard {
    int prev = -1; bool active = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) { active = (cudaSetDevice(dev) == cudaSuccess); }
    }
    ~DeviceGuard() { if (active) cudaSetDevice(prev); }
};

int ensure(lsp_ctx* h, void** ptr, size_t* have, size_t need) {
    if (need <= *have) return LSP_OK;
    if (*ptr) { cudaError_t e = cudaFree(*ptr); *ptr = nullptr; *have = 0; if (e != cudaSuccess) return cuda_fail(h, e); }
    need = align_up(need + need / 8, (size_t)1 << 20);
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, need);
    if (e != cudaSuccess) { h->last_cuda = (int)e; cudaGetLastError(); return LSP_ENOMEM; }
    *ptr = p; *have = need;
    return LSP_OK;
}

bool valid_K(int64_t K) { return K == 4 || K == 8 || K == 12 || K == 16 || K == 20 || K == 24 || K == 28 || K == 32; }

typedef void (*accum_fn)(const AccumParams);

struct KernelEntry { int K, rec; accum_fn fn; const char* name; int tile_z; int max_t; };   // tile_z = 0: pair-packed kernel

#define LSP_ENTRY(K, R, RN) { K, R, accum_kernel<K, R>, "accum_kernel<K=" #K "," RN ">", 0, 256 }
#define LSP_ENTRY_Z(K, TZ, MAXT, MINB) { K, REC_THREE_TERM_Z, accum_z_kernel<K, TZ, MAXT, MINB>, "accum_z_kernel<K=" #K ",three_term_z>", TZ, MAXT }
const KernelEntry g_kernels[] = {
    LSP_ENTRY(4,  REC_ROTATION, "rotation"),   LSP_ENTRY(4,  REC_THREE_TERM, "three_term"),
    LSP_ENTRY(8,  REC_ROTATION, "rotation"),   LSP_ENTRY(8,  REC_THREE_TERM, "three_term"),
    LSP_ENTRY(12, REC_ROTATION, "rotation"),   LSP_ENTRY(12, REC_THREE_TERM, "three_term"),
    LSP_ENTRY(16, REC_ROTATION, "rotation"),   LSP_ENTRY(16, REC_THREE_TERM, "three_term"),
    LSP_ENTRY(20, REC_ROTATION, "rotation"),   LSP_ENTRY(20, REC_THREE_TERM, "three_term"),
    LSP_ENTRY(24, REC_ROTATION, "rotation"),   LSP_ENTRY(24, REC_THREE_TERM, "three_term"),
    LSP_ENTRY_Z(4, 256, 256, 1), LSP_ENTRY_Z(8, 256, 256, 1), LSP_ENTRY_Z(12, 256, 256, 1), LSP_ENTRY_Z(16, 256, 256, 1),
    LSP_ENTRY_Z(20, 256, 256, 1), LSP_ENTRY_Z(24, 256, 256, 2), LSP_ENTRY_Z(28, 256, 128, 3), LSP_ENTRY_Z(32, 256, 128, 3),
};

const KernelEntry* find_kernel(int K, int rec) {
    for (const KernelEntry& e : g_kernels) if (e.K == K && e.rec == rec) return &e;
    return nullptr;
}

size_t accum_smem_bytes(const KernelEntry* ke, int T) {
    if (ke->tile_z) return (size_t)ke->tile_z * 24 + (size_t)T * (4 * ke->K + 1) * sizeof(float);
    return (size_t)3 * PAIRS * 16 + (size_t)4 * ke->K * T * sizeof(float);
}

// Launch plan: which (K, T), how many time splits.  Units of work = B * nfb * nsplit CTAs; the
// hardware block scheduler balances them over the SMs, so we want many more units than CTA slots.
Plan make_plan(const lsp_ctx* h, int64_t B, int64_t Nt, int64_t Nf) {
    Plan pl;
    PlanOverrides ov;
    ov.K = h->opt_K; ov.T = h->opt_T; ov.nsplit = h->opt_nsplit; ov.rec = h->opt_rec; ov.L = h->opt_coarse;
    const PlanChoice pc = plan_choose(h->sm_count, B, Nt, Nf, ov);
    pl.rec = pc.rec; pl.K = pc.K; pl.T = pc.T; pl.nfb = pc.nfb; pl.L = pc.L;
    pl.nsplit = pc.nsplit; pl.split_len = pc.split_len;
    int64_t flush = h->opt_flush ? h->opt_flush : 2048;
    pl.flush_tiles = (int)((flush + TILE - 1) / TILE);
    if (pl.flush_tiles < 1) pl.flush_tiles = 1;
    // pre-pass partition: contiguous chunks, at most MAX_PARTS blocks per series
    int64_t nparts = (Nt + 4095) / 4096;
    if (nparts > MAX_PARTS) nparts = MAX_PARTS;
    if (B >= 64 && nparts > 4) nparts = 4;
    pl.nparts = (int)nparts;
    pl.part_chunk = (Nt + nparts - 1) / nparts;
    pl.nparts = (int)((Nt + pl.part_chunk - 1) / pl.part_chunk);
    pl.launches = 4;
    return pl;
}

// Shared-time batch (t_stride = 0): XC, XS as one dense GEMM over all series, CC, CS once per frequency (lsp_shared_gemm.cuh).
int run_device_shared(lsp_ctx* h, const double* t, const float* x, int64_t x_stride,
                      int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                      float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, cudaStream_t st)
{
    Plan pl = make_plan(h, B, Nt, Nf);                    // pre-pass partition only
    int64_t nsplit = (Nt + SG_MAX_SPLIT - 1) / SG_MAX_SPLIT;
    int64_t gps = ((Nt + nsplit - 1) / nsplit + SG_KS - 1) / SG_KS;
    gps = (gps + SG_KPS - 1) / SG_KPS * SG_KPS;           // k-step groups per split: whole stages
    nsplit = (Nt + gps * SG_KS - 1) / (gps * SG_KS);
    const int64_t ng = nsplit * gps;
    const int64_t nmb = (B + SG_M - 1) / SG_M, nfb = (Nf + SG_F - 1) / SG_F;
    const int64_t x_row = (Nf + 3) / 4 * 4;
    if (nmb * nfb * nsplit > 2147483647LL || ng > 65535 || nsplit > 65535 || B > 65535) return LSP_EINVAL;
    pl.rec = REC_UMMA; pl.K = SG_F; pl.T = SG_THREADS; pl.nsplit = (int)nsplit; pl.nfb = (int)nfb; pl.L = 0;
    pl.split_len = gps * SG_KS; pl.launches = 7;
    pl.kernel_name = (nsplit == 1) ? "shared_gemm_kernel<tcgen05.m128n256.f16+e5m2corr,TMA-fed,shared-times,fused-finish>"
                                   : "shared_gemm_kernel<tcgen05.m128n256.f16+e5m2corr,TMA-fed,shared-times>";

    const size_t n_samp = (size_t)B * (size_t)Nt;
    size_t off = 0;
    const size_t o_recA = off;                            // (no per-sample records per series on this path)
    const size_t o_recB = off; off = align_up(off + (size_t)Nt * sizeof(ulonglong2), 256);   // phases of the one time vector
    const size_t o_xa = off;   off = align_up(off + (size_t)nmb * ng * SG_A_GROUP, 256);
    const size_t o_eb = off;   off = align_up(off + (size_t)nfb * ng * SG_B_GROUP, 256);
    const size_t o_wsv = off;  off = align_up(off + (size_t)nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    const bool fuse = (nsplit == 1);                      // one split: the GEMM's accumulators are the sums; steps 6-7 run in its epilogue
    const size_t o_wsx = off;  if (!fuse) off = align_up(off + (size_t)B * nsplit * 2 * (size_t)x_row * sizeof(float), 256);
    const size_t o_vc = off;   off = align_up(off + (size_t)4 * (size_t)Nf * sizeof(double), 256);
    const size_t o_vcf = off;  off = align_up(off + (size_t)Nf * sizeof(float4), 256);
    const size_t o_psum = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    const size_t o_pvar = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    const size_t o_peak = off; off = align_up(off + (size_t)B * sizeof(u64), 256);
    const size_t o_cnt = off;  off = align_up(off + (size_t)B * sizeof(unsigned), 256);
    int rc = ensure(h, &h->buf, &h->buf_bytes, off);
    if (rc != LSP_OK) return rc;
    char* base = static_cast<char*>(h->buf);
    float4* recA = reinterpret_cast<float4*>(base + o_recA);
    ulonglong2* recB = reinterpret_cast<ulonglong2*>(base + o_recB);
    unsigned char* xa = reinterpret_cast<unsigned char*>(base + o_xa);
    unsigned char* eb = reinterpret_cast<unsigned char*>(base + o_eb);
    float* ws_v = reinterpret_cast<float*>(base + o_wsv);
    float* ws_x = reinterpret_cast<float*>(base + o_wsx);
    double* vconst = reinterpret_cast<double*>(base + o_vc);
    float4* vconst_f = reinterpret_cast<float4*>(base + o_vcf);
    double* psum = reinterpret_cast<double*>(base + o_psum);
    double* pvar = reinterpret_cast<double*>(base + o_pvar);
    u64* peak64 = reinterpret_cast<u64*>(base + o_peak);
    unsigned* counter = reinterpret_cast<unsigned*>(base + o_cnt);

    const bool timing = h->opt_timing != 0;
    cudaEvent_t* ev = h->ev[h->timed_calls % TIMING_RING];
    if (timing) {
        for (int i = 0; i < 5; ++i)
            if (!ev[i]) LSP_CUDA(h, cudaEventCreate(&ev[i]));
        LSP_CUDA(h, cudaEventRecord(ev[0], st));
    }
    // steps 1-2 (per series: mean, variance, X; the phase records of series 0 serve all)
    dim3 gpre((unsigned)pl.nparts, (unsigned)B);
    const bool fused_pre = pl.nparts == 1;                // one block per series: step 1's sum inside the records kernel
    if (!fused_pre) {
        moments_kernel<<<gpre, 256, 0, st>>>(x, x_stride, Nt, pl.part_chunk, psum, peak64, counter);
        LSP_CUDA(h, cudaGetLastError());
    } else pl.launches -= 1;
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[1], st));
    if (fused_pre) records_kernel<true, true><<<gpre, 256, 0, st>>>(t, 0, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter);
    else records_kernel<true, false><<<gpre, 256, 0, st>>>(t, 0, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter);
    LSP_CUDA(h, cudaGetLastError());
    // step 3 for every (sample, frequency) once; CC, CS once per frequency
    shared_e_kernel<<<dim3((unsigned)nfb, (unsigned)ng), 256, 0, st>>>(recB, Nt, Nf, eb, (int)ng);
    LSP_CUDA(h, cudaGetLastError());
    shared_v_kernel<<<dim3((unsigned)((Nf + 7) / 8), (unsigned)nsplit), 256, 0, st>>>(recB, Nt, Nf, gps * SG_KS, ws_v);
    LSP_CUDA(h, cudaGetLastError());
    if (fuse) {
        shared_vconst_kernel<<<(unsigned)((Nf + 255) / 256), 256, 0, st>>>(ws_v, (int)nsplit, Nf, Nt, vconst, vconst_f);
        LSP_CUDA(h, cudaGetLastError());
    }
    shared_x_kernel<<<dim3((unsigned)nmb, (unsigned)ng), 256, 0, st>>>(x, x_stride, psum, pvar, pl.nparts, B, Nt, xa, (int)ng);
    LSP_CUDA(h, cudaGetLastError());
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[2], st));
    // steps 4-5: the contraction
    SharedGemmParams gp;
    gp.xa = xa; gp.eb = eb; gp.ws_x = ws_x; gp.B = B; gp.Nf = Nf; gp.x_row = x_row;
    gp.nmb = (int)nmb; gp.nfb = (int)nfb; gp.nsplit = (int)nsplit; gp.ng = (int)ng; gp.groups_per_split = (int)gps;
    gp.vconst = fuse ? vconst : nullptr; gp.vconst_f = vconst_f; gp.part_var = pvar; gp.P = P; gp.p_stride = p_stride;
    gp.peak_idx = peak_idx; gp.peak_val = peak_val; gp.peak64 = peak64; gp.counter = counter; gp.Nt = Nt; gp.nparts = pl.nparts;
    LSP_CUDA(h, cudaFuncSetAttribute(shared_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SG_SMEM));
    shared_gemm_kernel<<<(unsigned)(nmb * nfb * nsplit), SG_THREADS, SG_SMEM, st>>>(gp);
    LSP_CUDA(h, cudaGetLastError());
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[3], st));
    if (fuse) {                                           // steps 6-7 ran in the GEMM's epilogue
        if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
        h->plan = pl;
        return LSP_OK;
    }
    // steps 6-7
    FinishParams fp;
    fp.ws = ws_v; fp.part_var = pvar; fp.P = P; fp.p_stride = p_stride;
    fp.peak_idx = peak_idx; fp.peak_val = peak_val; fp.peak64 = peak64; fp.counter = counter;
    fp.Nt = Nt; fp.Nf = Nf; fp.nsplit = (int)nsplit; fp.nparts = pl.nparts;
    fp.cc_fix = 0.0; fp.x_scaled = 1; fp.ws1 = nullptr; fp.ws_x = ws_x; fp.x_row = x_row;
    const int64_t per_block = (int64_t)FIN_THREADS * FIN_FPT;
    dim3 gfin((unsigned)((Nf + per_block - 1) / per_block), (unsigned)B);
    finish_kernel<<<gfin, FIN_THREADS, 0, st>>>(fp);
    LSP_CUDA(h, cudaGetLastError());
    if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
    h->plan = pl;
    return LSP_OK;
}

int run_device(lsp_ctx* h,
               const double* t, int64_t t_stride, const float* x, int64_t x_stride,
               int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
               float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, cudaStream_t st, bool gls = false)
{
    if (t_stride == 0 && B > 1 && !gls && h->opt_shared != 1 && h->opt_rec == 0 && B <= 65535 &&
        (h->opt_shared == 2 || (B >= 16 && Nt >= 512)))
        return run_device_shared(h, t, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride, peak_idx, peak_val, st);
    Plan pl = make_plan(h, B, Nt, Nf);
    const bool umma = pl.rec == REC_UMMA;
    const bool mma = pl.rec == REC_MMA || umma;                      // tensor-core forms: X scaled to unit variance
    const KernelEntry* ke = mma ? nullptr : find_kernel(pl.K, pl.rec);
    if (!mma && (!ke || pl.T < 32 || pl.T > ke->max_t || (pl.T % 32) != 0)) return LSP_EINVAL;
    const bool umma_small = umma && pl.L < UM_L;          // 128 x L frequencies per CTA, two CTAs per SM
    pl.kernel_name = umma ? "accum_umma_kernel<tcgen05.m128n256k16.f16,hi+lo>"
                          : (mma ? "accum_mma_kernel<m16n8k16.f16,hi+lo>" : ke->name);
    const bool duo = umma_small && pl.L == 16 && B >= 2 && h->opt_duo != 1;   // batches: two series per CTA (lsp_accum_umma_duo.cuh)
    if (umma_small) pl.kernel_name = pl.L == 16 ? "accum_umma_small_kernel<tcgen05.m128n32k16.f16,hi+lo>"
                                   : (pl.L == 32 ? "accum_umma_small_kernel<tcgen05.m128n64k16.f16,hi+lo>"
                                                 : "accum_umma_small_kernel<tcgen05.m128n128k16.f16,hi+lo>");

    // one CTA sees all samples of its series in one drain window: steps 6-7 run in its epilogue, no workspace round trip
    const bool duo_fuse = duo && !gls && pl.nsplit == 1 && Nt <= (h->opt_flush ? h->opt_flush : 2048);
    if (duo) pl.kernel_name = duo_fuse ? "accum_umma_duo_kernel<tcgen05.m128n128k16.f16,hi+lo,2 series x 64 x 32,fused-finish>"
                                       : "accum_umma_duo_kernel<tcgen05.m128n128k16.f16,hi+lo,2 series x 64 x 32>";
    if (duo_fuse) pl.launches = 3;

    // workspace carve-up
    const size_t n_samp = (size_t)B * (size_t)Nt;
    size_t off = 0;
    const size_t o_recA = off; off = align_up(off + n_samp * sizeof(float4), 256);
    const size_t o_recB = off; off = align_up(off + n_samp * sizeof(ulonglong2), 256);
    const size_t o_ws = off;   off = align_up(off + (size_t)B * pl.nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    const size_t o_ws1 = off;  if (gls) off = align_up(off + (size_t)B * pl.nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    const size_t o_recA1 = off; if (gls) off = align_up(off + n_samp * sizeof(float4), 256);
    const size_t o_psum = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    const size_t o_pvar = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    const size_t o_peak = off; off = align_up(off + (size_t)B * sizeof(u64), 256);
    const size_t o_cnt = off;  off = align_up(off + (size_t)B * sizeof(unsigned), 256);
    // tcgen05 form: the coarse operand B comes from a table when several frequency blocks share it (lsp_accum_umma_tab.cuh)
    const int64_t tab_series = (t_stride == 0) ? 1 : B;
    const int64_t tab_groups = (Nt + UM_KS - 1) / UM_KS + UT_KPS;
    const size_t tab_bytes = (size_t)tab_series * (size_t)tab_groups * UT_GROUP_BYTES;
    const bool use_tab = umma && !umma_small && h->opt_btable != 1 &&
                         (h->opt_btable == 2 || (pl.nfb >= 3 && tab_bytes <= ((size_t)12 << 30)));
    const size_t o_tab = off;  if (use_tab) off = align_up(off + tab_bytes, 256);
    const bool corr8 = use_tab && h->opt_corr != 1;       // correction products as one 8-bit MMA (default) or two fp16 MMAs
    const bool pair = corr8 && h->opt_pair != 1;          // CTA pairs (cta_group::2) share one B tile: lsp_accum_umma_pair.cuh
    const bool pair2 = pair && h->opt_pair != 2;          // ... and share the GENERATED operand instead: lsp_accum_umma_pair2.cuh (default)
    if (pair) pl.nfb = (pl.nfb + 1) & ~1;                 // a pair = two adjacent frequency blocks; an odd count gets one masked block
    if (use_tab) {
        pl.kernel_name = corr8 ? "accum_umma_tab_kernel<tcgen05.m128n256.f16+e5m2corr,B-table>"
                               : "accum_umma_tab_kernel<tcgen05.m128n256k16.f16,hi+lo,B-table>";
        if (pair) pl.kernel_name = pair2 ? "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16+e5m2corr,fine-table>"
                                         : "accum_umma_pair_kernel<tcgen05.cta_group2.m256n256.f16+e5m2corr,B-table>";
        pl.launches = 5;
        pl.mma_slots = corr8 ? 3 : 4;
    }
    if (gls) pl.launches += 2;                            // unit records + second accumulate pass
    int rc = ensure(h, &h->buf, &h->buf_bytes, off);
    if (rc != LSP_OK) return rc;
    char* base = static_cast<char*>(h->buf);
    float4* recA = reinterpret_cast<float4*>(base + o_recA);
    ulonglong2* recB = reinterpret_cast<ulonglong2*>(base + o_recB);
    float* ws = reinterpret_cast<float*>(base + o_ws);
    float* ws1 = gls ? reinterpret_cast<float*>(base + o_ws1) : nullptr;          // unit-weight pass: sum cos, sum sin
    float4* recA1 = gls ? reinterpret_cast<float4*>(base + o_recA1) : nullptr;
    double* psum = reinterpret_cast<double*>(base + o_psum);
    double* pvar = reinterpret_cast<double*>(base + o_pvar);
    u64* peak64 = reinterpret_cast<u64*>(base + o_peak);
    unsigned* counter = reinterpret_cast<unsigned*>(base + o_cnt);

    if (B > 65535) return LSP_EINVAL;                     // grid.y limit of the pre-pass / finish kernels

    const bool timing = h->opt_timing != 0;
    cudaEvent_t* ev = h->ev[h->timed_calls % TIMING_RING];
    if (timing) {
        for (int i = 0; i < 5; ++i)
            if (!ev[i]) LSP_CUDA(h, cudaEventCreate(&ev[i]));
        LSP_CUDA(h, cudaEventRecord(ev[0], st));
    }

    // steps 1-2
    dim3 gpre((unsigned)pl.nparts, (unsigned)B);
    const bool fused_pre = pl.nparts == 1;                // one block per series: step 1's sum inside the records kernel
    if (!fused_pre) {
        moments_kernel<<<gpre, 256, 0, st>>>(x, x_stride, Nt, pl.part_chunk, psum, peak64, counter);
        LSP_CUDA(h, cudaGetLastError());
    } else pl.launches -= 1;
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[1], st));
    if (fused_pre) records_kernel<false, true><<<gpre, 256, 0, st>>>(t, t_stride, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter);
    else records_kernel<false, false><<<gpre, 256, 0, st>>>(t, t_stride, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter);
    LSP_CUDA(h, cudaGetLastError());
    if (gls) {
        unit_records_kernel<<<(unsigned)((n_samp + 255) / 256), 256, 0, st>>>(recA, recA1, (int64_t)n_samp);
        LSP_CUDA(h, cudaGetLastError());
    }
    unsigned char* btable = reinterpret_cast<unsigned char*>(base + o_tab);
    if (use_tab) {
        if (tab_groups > 2147483647LL) return LSP_EINVAL;
        dim3 gtab((unsigned)tab_groups, (unsigned)tab_series);
        if (pair2) umma_ftable_pair_kernel<<<gtab, 512, 0, st>>>(recB, Nt, Nt, btable, (int64_t)tab_groups * UP_GROUP_BYTES, (int64_t)tab_groups * UT_GROUP_BYTES);
        else if (pair) umma_btable_pair_kernel<<<gtab, 256, 0, st>>>(recB, Nt, Nt, btable, (int64_t)tab_groups * UP_GROUP_BYTES, (int64_t)tab_groups * UT_GROUP_BYTES);
        else if (corr8) umma_btable_kernel<true><<<gtab, 256, 0, st>>>(recB, Nt, Nt, btable, tab_groups, (int64_t)tab_groups * UT_GROUP_BYTES);
        else umma_btable_kernel<false><<<gtab, 256, 0, st>>>(recB, Nt, Nt, btable, tab_groups, (int64_t)tab_groups * UT_GROUP_BYTES);
        LSP_CUDA(h, cudaGetLastError());
    }

    if (timing) LSP_CUDA(h, cudaEventRecord(ev[2], st));

    // steps 3-5
    const int64_t units = (duo ? (B + 1) / 2 : B) * (int64_t)pl.nsplit * pl.nfb;
    if (units > 2147483647LL) return LSP_EINVAL;
    // (generalised periodogram: a second pass with unit weights gives sum cos, sum sin in ws1)
    for (int pass = 0; pass < (gls ? 2 : 1); ++pass) {
    const float4* rA = pass ? recA1 : recA;
    float* wsp = pass ? ws1 : ws;
    if (umma) {
        UmmaParams up;
        up.recA = rA; up.recB = recB; up.part_var = pvar; up.ws = wsp; up.Nt = Nt; up.Nf = Nf;
        up.split_len = pl.split_len; up.nsplit = pl.nsplit; up.nfb = pl.nfb; up.nparts = pl.nparts;
        // drain interval of D_W: 2,048 samples; 4,096 for the pair2 form, whose drain adds the expected truncation loss back
        // (measured max error of max P at 2,048 / 4,096 / 8,192 samples: C3 5e-6 / 9e-6 / 2.2e-5, C5 4e-6 / 6e-6 / 1.1e-5, P0 9e-6 / 1.9e-5 / 3.8e-5)
        up.flush_ksteps = (int)((h->opt_flush ? h->opt_flush : (pair2 ? 4096 : 2048)) + UM_KS - 1) / UM_KS;
        up.trunc_ulps = pair2 ? 0.45f : 0.f;
        up.unit_x = pass;
        if (duo) {
            UmmaDuoParams dp;
            dp.u = up; dp.B = B;
            dp.fuse = duo_fuse ? 1 : 0; dp.P = P; dp.p_stride = p_stride;
            dp.peak_idx = peak_idx; dp.peak_val = peak_val; dp.peak64 = peak64; dp.counter = counter;
            LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_duo_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UD_SMEM));
            accum_umma_duo_kernel<<<(unsigned)units, US_THREADS, UD_SMEM, st>>>(dp);
        } else if (umma_small) {
#define LSP_LAUNCH_SMALL(LL, NS, MINB) do { \
            LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_small_kernel<LL, NS, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UmmaSmall<LL, NS>::SMEM)); \
            accum_umma_small_kernel<LL, NS, MINB><<<(unsigned)units, US_THREADS, UmmaSmall<LL, NS>::SMEM, st>>>(up); } while (0)
            if (pl.L == 16) LSP_LAUNCH_SMALL(16, 4, 3);
            else if (pl.L == 32) LSP_LAUNCH_SMALL(32, 4, 2);
            else if (pl.L == 64) LSP_LAUNCH_SMALL(64, 4, 2);
            else return LSP_EINVAL;
#undef LSP_LAUNCH_SMALL
        } else if (use_tab) {
            UmmaTabParams tp;
            tp.u = up; tp.btable = btable; tp.ngroups = tab_groups;
            tp.table_stride = (tab_series == 1) ? 0 : (int64_t)tab_groups * UT_GROUP_BYTES;
            if (pair) {
                UmmaPairParams pp;
                pp.u = up; pp.btable = btable; pp.half_stride = (int64_t)tab_groups * UP_GROUP_BYTES;
                pp.table_stride = tp.table_stride;
                LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UP_SMEM));
                LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_pair2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)U2_SMEM));
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3((unsigned)units); cfg.blockDim = dim3(pair2 ? U2_THREADS : UM_THREADS); cfg.dynamicSmemBytes = pair2 ? U2_SMEM : UP_SMEM; cfg.stream = st;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                if (pair2) LSP_CUDA(h, cudaLaunchKernelEx(&cfg, accum_umma_pair2_kernel, pp));
                else LSP_CUDA(h, cudaLaunchKernelEx(&cfg, accum_umma_pair_kernel, pp));
            } else if (corr8) {
                LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_tab_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UT_SMEM));
                accum_umma_tab_kernel<true><<<(unsigned)units, UM_THREADS, UT_SMEM, st>>>(tp);
            } else {
                LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_tab_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UT_SMEM));
                accum_umma_tab_kernel<false><<<(unsigned)units, UM_THREADS, UT_SMEM, st>>>(tp);
            }
        } else {
            LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UM_SMEM));
            accum_umma_kernel<<<(unsigned)units, UM_THREADS, UM_SMEM, st>>>(up);
        }
    } else if (mma) {
        MmaParams mp;
        mp.recA = rA; mp.recB = recB; mp.part_var = pvar; mp.ws = wsp; mp.Nt = Nt; mp.Nf = Nf;
        mp.split_len = pl.split_len; mp.nsplit = pl.nsplit; mp.nfb = pl.nfb; mp.nparts = pl.nparts; mp.unit_x = pass;
        LSP_CUDA(h, cudaFuncSetAttribute(accum_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MMA_SMEM));
        accum_mma_kernel<<<(unsigned)units, MMA_WARPS * 32, MMA_SMEM, st>>>(mp);
    } else {
        AccumParams ap;
        ap.recA = rA; ap.recB = recB; ap.ws = wsp; ap.Nt = Nt; ap.Nf = Nf;
        ap.split_len = pl.split_len; ap.nsplit = pl.nsplit; ap.nfb = pl.nfb; ap.flush_tiles = pl.flush_tiles;
        const size_t smem = accum_smem_bytes(ke, pl.T);
        LSP_CUDA(h, cudaFuncSetAttribute(ke->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ke->fn<<<(unsigned)units, pl.T, smem, st>>>(ap);
    }
    LSP_CUDA(h, cudaGetLastError());
    }
    LSP_CUDA(h, cudaGetLastError());

    if (timing) LSP_CUDA(h, cudaEventRecord(ev[3], st));

    if (duo_fuse) {
        if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
        h->plan = pl;
        return LSP_OK;
    }
    // steps 6-7
    FinishParams fp;
    fp.ws = ws; fp.part_var = pvar; fp.P = P; fp.p_stride = p_stride;
    fp.peak_idx = peak_idx; fp.peak_val = peak_val; fp.peak64 = peak64; fp.counter = counter;
    fp.Nt = Nt; fp.Nf = Nf; fp.nsplit = pl.nsplit; fp.nparts = pl.nparts;
    fp.cc_fix = (!mma && ke->tile_z == 0 && (Nt & 1)) ? 0.5 : 0.0;   // phantom partner of an odd last sample (pair-packed only)
    fp.x_scaled = mma ? 1 : 0;
    fp.ws1 = ws1;
    fp.ws_x = nullptr; fp.x_row = 0;
    const int64_t per_block = (int64_t)FIN_THREADS * FIN_FPT;
    dim3 gfin((unsigned)((Nf + per_block - 1) / per_block), (unsigned)B);
    finish_kernel<<<gfin, FIN_THREADS, 0, st>>>(fp);
    LSP_CUDA(h, cudaGetLastError());
    if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }

    h->plan = pl;
    return LSP_OK;
}

bool bad_grid(double f_min, double df) {
    return !(std::isfinite(f_min) && std::isfinite(df)) || f_min < 0.0 || df < 0.0;
}

}  // namespace

// ------------------------------------------------------------------------------------------ C ABI
extern "C" {

int lsp_create(lsp_handle* out, int device)
{
    if (!out) return LSP_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return LSP_ECUDA; }
    if (device < 0) { if (cudaGetDevice(&device) != cudaSuccess) return LSP_ECUDA; }
    if (device >= ndev) return LSP_EINVAL;
    lsp_ctx* h = new (std::nothrow) lsp_ctx();
    if (!h) return LSP_ENOMEM;
    h->device = device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete h; return LSP_ECUDA; }
    h->sm_count = prop.multiProcessorCount;
    if (prop.major < 10) {                                // sm_100a SASS only: fail loudly elsewhere
        delete h;
        return LSP_ECUDA;
    }
    *out = h;
    return LSP_OK;
}

int lsp_destroy(lsp_handle h)
{
    if (!h) return LSP_OK;
    DeviceGuard g(h->device);
    cudaDeviceSynchronize();
    if (h->buf) cudaFree(h->buf);
    if (h->stage) cudaFree(h->stage);
    for (int r = 0; r < TIMING_RING; ++r)
        for (int i = 0; i < 5; ++i) if (h->ev[r][i]) cudaEventDestroy(h->ev[r][i]);
    delete h;
    return LSP_OK;
}

int lsp_set_param(lsp_handle h, int key, int64_t value)
{
    if (!h || value < 0) return LSP_EINVAL;
    switch (key) {
        case LSP_PARAM_K:          if (value && !valid_K(value)) return LSP_EINVAL; h->opt_K = value; break;
        case LSP_PARAM_THREADS:    if (value && (value < 32 || value > 256 || value % 32)) return LSP_EINVAL; h->opt_T = value; break;
        case LSP_PARAM_NSPLIT:     h->opt_nsplit = value; break;
        case LSP_PARAM_RECURRENCE: if (value > 5) return LSP_EINVAL; h->opt_rec = value; break;
        case LSP_PARAM_FLUSH:      h->opt_flush = value; break;
        case LSP_PARAM_TIMING:     if (value > 1) return LSP_EINVAL; h->opt_timing = value; break;
        case LSP_PARAM_BTABLE:     if (value > 2) return LSP_EINVAL; h->opt_btable = value; break;
        case LSP_PARAM_COARSE:     if (value && value != 16 && value != 32 && value != 64 && value != 128) return LSP_EINVAL; h->opt_coarse = value; break;
        case LSP_PARAM_CORR:       if (value > 2) return LSP_EINVAL; h->opt_corr = value; break;
        case LSP_PARAM_PAIR:       if (value > 3) return LSP_EINVAL; h->opt_pair = value; break;
        case LSP_PARAM_SHARED:     if (value > 2) return LSP_EINVAL; h->opt_shared = value; break;
        case LSP_PARAM_DUO:        if (value > 2) return LSP_EINVAL; h->opt_duo = value; break;
        default: return LSP_EINVAL;
    }
    return LSP_OK;
}

int lsp_get_param(lsp_handle h, int key, int64_t* value)
{
    if (!h || !value) return LSP_EINVAL;
    switch (key) {
        case LSP_PARAM_K:          *value = h->opt_K; break;
        case LSP_PARAM_THREADS:    *value = h->opt_T; break;
        case LSP_PARAM_NSPLIT:     *value = h->opt_nsplit; break;
        case LSP_PARAM_RECURRENCE: *value = h->opt_rec; break;
        case LSP_PARAM_FLUSH:      *value = h->opt_flush; break;
        case LSP_PARAM_TIMING:     *value = h->opt_timing; break;
        case LSP_PARAM_BTABLE:     *value = h->opt_btable; break;
        case LSP_PARAM_COARSE:     *value = h->opt_coarse; break;
        case LSP_PARAM_CORR:       *value = h->opt_corr; break;
        case LSP_PARAM_PAIR:       *value = h->opt_pair; break;
        case LSP_PARAM_SHARED:     *value = h->opt_shared; break;
        case LSP_PARAM_DUO:        *value = h->opt_duo; break;
        default: return LSP_EINVAL;
    }
    return LSP_OK;
}

int lsp_call_timing(lsp_handle h, int calls_back, float ms[4])
{
    if (!h || !ms || calls_back < 0) return LSP_EINVAL;
    if ((uint64_t)calls_back >= h->timed_calls || calls_back >= TIMING_RING) return LSP_EINVAL;
    DeviceGuard g(h->device);
    cudaEvent_t* ev = h->ev[(h->timed_calls - 1 - (uint64_t)calls_back) % TIMING_RING];
    LSP_CUDA(h, cudaEventSynchronize(ev[4]));
    for (int i = 0; i < 4; ++i) LSP_CUDA(h, cudaEventElapsedTime(&ms[i], ev[i], ev[i + 1]));
    return LSP_OK;
}

int lsp_last_timing(lsp_handle h, float ms[4]) { return lsp_call_timing(h, 0, ms); }

int lsp_plan_query(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int64_t out[8])
{
    if (!out || sm_count < 1 || B < 1 || Nt < 2 || Nf < 1) return LSP_EINVAL;
    const PlanChoice pc = plan_choose(sm_count, B, Nt, Nf, PlanOverrides());
    out[0] = pc.K; out[1] = pc.T; out[2] = pc.nsplit; out[3] = pc.rec;
    out[4] = pc.nfb; out[5] = pc.split_len; out[6] = pc.ctas_per_sm;
    out[7] = (int64_t)(pc.score * 1e6);
    return LSP_OK;
}

int lsp_plan_query_form(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int recurrence, int64_t out[8])
{
    if (!out || sm_count < 1 || B < 1 || Nt < 2 || Nf < 1 || recurrence < 0 || recurrence > 5) return LSP_EINVAL;
    PlanOverrides ov;
    ov.rec = recurrence;
    const PlanChoice pc = plan_choose(sm_count, B, Nt, Nf, ov);
    out[0] = pc.K; out[1] = pc.T; out[2] = pc.nsplit; out[3] = pc.rec;
    out[4] = pc.nfb; out[5] = pc.split_len; out[6] = pc.ctas_per_sm;
    out[7] = (int64_t)plan_est_cycles(sm_count, B, Nt, Nf, pc);
    return LSP_OK;
}

int lsp_periodogram_batched(lsp_handle h,
                            const double* t, int64_t t_stride, const float* x, int64_t x_stride,
                            int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                            float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, void* stream)
{
    if (!h || !t || !x) return LSP_EINVAL;
    if (B < 1 || Nt < 2 || Nf < 1 || Nt > 2000000000LL || Nf > 2000000000LL) return LSP_EINVAL;
    if (bad_grid(f_min, df)) return LSP_EINVAL;
    if ((peak_idx == nullptr) != (peak_val == nullptr)) return LSP_EINVAL;
    if (!P && !peak_idx) return LSP_EINVAL;
    if (B > 1) {
        if (t_stride != 0 && std::llabs(t_stride) < Nt) return LSP_EINVAL;
        if (std::llabs(x_stride) < Nt) return LSP_EINVAL;
        if (P && std::llabs(p_stride) < Nf) return LSP_EINVAL;
    }
    DeviceGuard g(h->device);
    return run_device(h, t, t_stride, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride,
                      peak_idx, peak_val, static_cast<cudaStream_t>(stream));
}

int lsp_periodogram_gls_batched(lsp_handle h,
                                const double* t, int64_t t_stride, const float* x, int64_t x_stride,
                                int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                                float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, void* stream)
{
    if (!h || !t || !x) return LSP_EINVAL;
    if (B < 1 || Nt < 4 || Nf < 1 || Nt > 2000000000LL || Nf > 2000000000LL) return LSP_EINVAL;
    if (bad_grid(f_min, df)) return LSP_EINVAL;
    if ((peak_idx == nullptr) != (peak_val == nullptr)) return LSP_EINVAL;
    if (!P && !peak_idx) return LSP_EINVAL;
    if (B > 1) {
        if (t_stride != 0 && std::llabs(t_stride) < Nt) return LSP_EINVAL;
        if (std::llabs(x_stride) < Nt) return LSP_EINVAL;
        if (P && std::llabs(p_stride) < Nf) return LSP_EINVAL;
    }
    DeviceGuard g(h->device);
    return run_device(h, t, t_stride, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride,
                      peak_idx, peak_val, static_cast<cudaStream_t>(stream), true);
}

int lsp_periodogram_gls(lsp_handle h, const double* t, const float* x, int64_t Nt,
                        double f_min, double df, int64_t Nf, float* P, void* stream)
{
    if (!P) return LSP_EINVAL;
    return lsp_periodogram_gls_batched(h, t, Nt, x, Nt, 1, Nt, f_min, df, Nf, P, Nf, nullptr, nullptr, stream);
}

int lsp_periodogram(lsp_handle h, const double* t, const float* x, int64_t Nt,
                    double f_min, double df, int64_t Nf, float* P, void* stream)
{
    if (!P) return LSP_EINVAL;
    return lsp_periodogram_batched(h, t, Nt, x, Nt, 1, Nt, f_min, df, Nf, P, Nf, nullptr, nullptr, stream);
}

int lsp_periodogram_batched_host(lsp_handle h, const double* t, int share_t, const float* x,
                                 int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                                 float* P, int32_t* peak_idx, float* peak_val, void* stream)
{
    if (!h || !t || !x) return LSP_EINVAL;
    if (B < 1 || Nt < 2 || Nf < 1 || Nt > 2000000000LL || Nf > 2000000000LL) return LSP_EINVAL;
    if (bad_grid(f_min, df)) return LSP_EINVAL;
    if ((peak_idx == nullptr) != (peak_val == nullptr)) return LSP_EINVAL;
    if (!P && !peak_idx) return LSP_EINVAL;
    DeviceGuard g(h->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nt_t = (size_t)(share_t ? 1 : B) * (size_t)Nt;
    const size_t nt_x = (size_t)B * (size_t)Nt;
    size_t off = 0;
    const size_t o_t = off; off = align_up(off + nt_t * sizeof(double), 256);
    const size_t o_x = off; off = align_up(off + nt_x * sizeof(float), 256);
    const size_t o_P = off; off = align_up(off + (P ? (size_t)B * (size_t)Nf * sizeof(float) : 0), 256);
    const size_t o_pi = off; off = align_up(off + (size_t)B * sizeof(int32_t), 256);
    const size_t o_pv = off; off = align_up(off + (size_t)B * sizeof(float), 256);
    int rc = ensure(h, &h->stage, &h->stage_bytes, off);
    if (rc != LSP_OK) return rc;
    char* base = static_cast<char*>(h->stage);
    double* d_t = reinterpret_cast<double*>(base + o_t);
    float* d_x = reinterpret_cast<float*>(base + o_x);
    float* d_P = P ? reinterpret_cast<float*>(base + o_P) : nullptr;
    int32_t* d_pi = peak_idx ? reinterpret_cast<int32_t*>(base + o_pi) : nullptr;
    float* d_pv = peak_val ? reinterpret_cast<float*>(base + o_pv) : nullptr;
    LSP_CUDA(h, cudaMemcpyAsync(d_t, t, nt_t * sizeof(double), cudaMemcpyHostToDevice, st));
    LSP_CUDA(h, cudaMemcpyAsync(d_x, x, nt_x * sizeof(float), cudaMemcpyHostToDevice, st));
    rc = run_device(h, d_t, share_t ? 0 : Nt, d_x, Nt, B, Nt, f_min, df, Nf, d_P, Nf, d_pi, d_pv, st);
    if (rc != LSP_OK) return rc;
    if (P) LSP_CUDA(h, cudaMemcpyAsync(P, d_P, (size_t)B * (size_t)Nf * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (peak_idx) {
        LSP_CUDA(h, cudaMemcpyAsync(peak_idx, d_pi, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(h, cudaMemcpyAsync(peak_val, d_pv, (size_t)B * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    LSP_CUDA(h, cudaStreamSynchronize(st));
    return LSP_OK;
}

int lsp_periodogram_host(lsp_handle h, const double* t, const float* x, int64_t Nt,
                         double f_min, double df, int64_t Nf, float* P, void* stream)
{
    if (!P) return LSP_EINVAL;
    return lsp_periodogram_batched_host(h, t, 0, x, 1, Nt, f_min, df, Nf, P, nullptr, nullptr, stream);
}

int lsp_false_alarm(lsp_handle h, const float* P, int64_t n, int64_t Nt, double N_ind, float* Q, void* stream)
{
    if (!h || !P || !Q || n < 1 || Nt < 4 || !(N_ind >= 1.0) || !std::isfinite(N_ind)) return LSP_EINVAL;
    DeviceGuard g(h->device);
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 2147483647LL) return LSP_EINVAL;
    fap_kernel<<<(unsigned)blocks, 256, 0, static_cast<cudaStream_t>(stream)>>>(P, n, (double)Nt, N_ind, Q);
    LSP_CUDA(h, cudaGetLastError());
    return LSP_OK;
}

int lsp_last_plan(lsp_handle h, int64_t out[8])
{
    if (!h || !out) return LSP_EINVAL;
    const Plan& p = h->plan;
    out[0] = p.K; out[1] = p.T; out[2] = p.nsplit; out[3] = p.rec;
    out[4] = p.nfb; out[5] = p.split_len; out[6] = p.launches;
    out[7] = (p.rec == REC_ROTATION) ? 8 : ((p.rec == REC_MMA || p.rec == REC_UMMA) ? 0 : 6);   // 0: tensor-core form (16 tensor FLOP per term)
    return LSP_OK;
}

const char* lsp_last_kernel_name(lsp_handle h) { return h ? h->plan.kernel_name : ""; }

int lsp_last_cuda_error(lsp_handle h) { return h ? h->last_cuda : 0; }

const char* lsp_status_string(int status)
{
    switch (status) {
        case LSP_OK:     return "ok";
        case LSP_EINVAL: return "invalid argument";
        case LSP_ECUDA:  return "CUDA runtime error (or no sm_100 device)";
        case LSP_ENOMEM: return "device workspace allocation failed";
        default:         return "unknown status";
    }
}

const char* lsp_version(void) { return "lsp_b200 0.1 (sm_100a)"; }

}  // extern "C"
