// lsp.cu -- host side of the C ABI declared in include/lsp.h: argument checks, launch plan,
// workspace, and the enqueues (moments -> records -> [table ->] accumulate -> finish).
// No CPU arithmetic on the data path: every step of SURVEY.md section 8(a) runs in a kernel.
#include "../../include/lsp.h"
#include "lsp_common.cuh"
#include "lsp_prepass.cuh"
#include "lsp_accum_z.cuh"
#include "lsp_tc.cuh"
#include "lsp_accum_umma_pair2.cuh"
#include "lsp_accum_umma_small.cuh"
#include "lsp_accum_umma_duo.cuh"
#include "lsp_shared_gemm.cuh"
#include "lsp_finish.cuh"
#include "lsp_fap.cuh"
#include "lsp_probe.cuh"
#include "lsp_plan.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <new>

using namespace lsp;

namespace {

struct Plan {
    int K = 0, T = 0, nsplit = 0, pipe = 0, nfb = 0, flush_tiles = 0, nparts = 0, launches = 0, L = 0, nchunks = 1;
    bool fused_pre = false;
    int64_t split_len = 0, part_chunk = 0, chunk_len = 0;
    const char* kernel_name = "";
};

}  // namespace

constexpr int HOST_PIPE_CHUNKS = 4;        // host-buffer batches: series chunks whose copies overlap the compute of their neighbours
constexpr int TIMING_RING = 64;
constexpr int TIMING_MAX_CHUNKS = 16;      // per-chunk accumulate events (more chunks: the accumulate bracket includes the later table pre-passes)

struct lsp_ctx {
    int device = 0;
    int sm_count = 148;
    int last_cuda = 0;
    // tunables (0 = automatic)
    int64_t opt_K = 0, opt_T = 0, opt_nsplit = 0, opt_pipe = 0, opt_flush = 0, opt_timing = 0, opt_table_mb = 0, opt_coarse = 0, opt_trunc = 0, opt_shared = 0, opt_pdl = 0, opt_corr = 0, opt_refine = 0, opt_order = 0;
    cudaEvent_t ev[TIMING_RING][5] = {};                  // ring of per-call event sets (LSP_PARAM_TIMING)
    cudaEvent_t evc[TIMING_RING][2 * TIMING_MAX_CHUNKS] = {};   // accumulate launches of a chunked call, begin / end per chunk
    int ev_chunks[TIMING_RING] = {};
    uint64_t timed_calls = 0;
    // workspace
    void* buf = nullptr;
    size_t buf_bytes = 0;
    void* refine_buf = nullptr;                           // list of ill-conditioned (series, frequency) pairs left by the fused epilogues (lsp_refine.cuh)
    // staging for the host-pointer entry points; copy streams and events of the pipelined batch form
    void* stage = nullptr;
    size_t stage_bytes = 0;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    int last_host_chunks = 0;
    cudaEvent_t ev_pipe[2 * HOST_PIPE_CHUNKS + 1] = {};
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

// Grow *ptr to `need` bytes.  The new buffer is allocated BEFORE the old one is released, so a failed allocation
// (LSP_ENOMEM) leaves the handle with the workspace it had.  cudaFree waits for work that still uses the old buffer.
int ensure(lsp_ctx* h, void** ptr, size_t* have, size_t need) {
    if (need <= *have) return LSP_OK;
    need = align_up(need + need / 8, (size_t)1 << 20);
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, need);
    if (e != cudaSuccess && *ptr) {                      // not enough room for both: the old contents are scratch, so retry after freeing
        cudaGetLastError();
        void* old = *ptr; const size_t old_bytes = *have;
        if (cudaFree(old) == cudaSuccess) {
            *ptr = nullptr; *have = 0;
            e = cudaMalloc(&p, need);
            if (e != cudaSuccess) {                      // put back what the handle had
                cudaGetLastError();
                void* back = nullptr;
                if (cudaMalloc(&back, old_bytes) == cudaSuccess) { *ptr = back; *have = old_bytes; } else cudaGetLastError();
                h->last_cuda = (int)e;
                return LSP_ENOMEM;
            }
            *ptr = p; *have = need;
            return LSP_OK;
        }
    }
    if (e != cudaSuccess) { h->last_cuda = (int)e; cudaGetLastError(); return LSP_ENOMEM; }
    if (*ptr) { cudaError_t f = cudaFree(*ptr); if (f != cudaSuccess) { cudaFree(p); return cuda_fail(h, f); } }
    *ptr = p; *have = need;
    return LSP_OK;
}

typedef void (*accum_fn)(const AccumParams);

struct KernelEntry { int K; accum_fn fn, fn_weighted, fn_direct, fn_gls, fn_gls_weighted, fn_gls_direct; const char* name; const char* name_weighted;
                     const char* name_gls; const char* name_gls_weighted; int max_t; };

constexpr int GLS_FUSED_MAX_K = 20;       // FP32 form, generalised periodogram in one pass (accum_z_kernel<..., GLS>): 2 K more registers per thread
#define LSP_ENTRY_Z(K, MAXT, MINB) { K, accum_z_kernel<K, MAXT, MINB>, accum_z_kernel<K, MAXT, MINB, true>, accum_z_kernel<K, MAXT, MINB, false, true>, \
                                     nullptr, nullptr, nullptr, \
                                     "accum_z_kernel<K=" #K ",fp32,three-term>", "accum_z_kernel<K=" #K ",fp32,three-term,weighted>", "", "", MAXT }
#define LSP_ENTRY_ZG(K, MAXT, MINB) { K, accum_z_kernel<K, MAXT, MINB>, accum_z_kernel<K, MAXT, MINB, true>, accum_z_kernel<K, MAXT, MINB, false, true>, \
                                     accum_z_kernel<K, MAXT, MINB, false, false, true>, accum_z_kernel<K, MAXT, MINB, true, false, true>, \
                                     accum_z_kernel<K, MAXT, MINB, false, true, true>, \
                                     "accum_z_kernel<K=" #K ",fp32,three-term>", "accum_z_kernel<K=" #K ",fp32,three-term,weighted>", \
                                     "accum_z_kernel<K=" #K ",fp32,three-term,generalised one-pass>", "accum_z_kernel<K=" #K ",fp32,three-term,generalised one-pass,weighted>", MAXT }
const KernelEntry g_kernels[] = {
    LSP_ENTRY_ZG(4, 256, 1), LSP_ENTRY_ZG(8, 256, 1), LSP_ENTRY_ZG(12, 256, 1), LSP_ENTRY_ZG(16, 256, 1),
    LSP_ENTRY_ZG(20, 256, 1), LSP_ENTRY_Z(24, 256, 2), LSP_ENTRY_Z(28, 128, 3), LSP_ENTRY_Z(32, 128, 3),
};
const KernelEntry* find_kernel(int K) {
    for (const KernelEntry& e : g_kernels) if (e.K == K) return &e;
    return nullptr;
}

size_t accum_smem_bytes(const KernelEntry* ke, int T, bool weighted, bool direct, bool gls_fused = false) {
    return (size_t)TILE_Z * (weighted ? 32 : 24) + (direct ? 0 : (size_t)T * ((gls_fused ? 6 : 4) * ke->K + 1) * sizeof(float));
}

// Launch plan: which form and tile, how many time splits (and chunks).  Units of work = B * nfb * nsplit CTAs; the
// hardware block scheduler balances them over the SMs, so we want many more units than CTA slots.
Plan make_plan(const lsp_ctx* h, int64_t B, int64_t Nt, int64_t Nf, int64_t table_series, int force_pipe = 0, int max_K = 32)
{
    Plan pl;
    PlanOverrides ov;
    ov.max_K = max_K;
    ov.K = h->opt_K; ov.T = h->opt_T; ov.nsplit = h->opt_nsplit; ov.pipe = force_pipe ? force_pipe : h->opt_pipe; ov.L = h->opt_coarse;
    ov.table_budget = h->opt_table_mb ? (h->opt_table_mb << 20) : 0; ov.table_series = table_series;
    const PlanChoice pc = plan_choose(h->sm_count, B, Nt, Nf, ov);
    pl.pipe = pc.pipe; pl.K = pc.K; pl.T = pc.T; pl.nfb = pc.nfb; pl.L = pc.L;
    pl.nsplit = pc.nsplit; pl.split_len = pc.split_len; pl.nchunks = pc.nchunks; pl.chunk_len = pc.chunk_len;
    const int64_t flush = h->opt_flush ? h->opt_flush : 2048;
    pl.flush_tiles = (int)((flush + TILE_Z - 1) / TILE_Z);
    if (pl.flush_tiles < 1) pl.flush_tiles = 1;
    // pre-pass partition: contiguous chunks, at most MAX_PARTS blocks per series
    int64_t nparts = (Nt + 4095) / 4096;
    if (nparts > MAX_PARTS) nparts = MAX_PARTS;
    if (B >= 64 && nparts > 4) nparts = 4;
    pl.fused_pre = Nt <= 16384;                           // short series: every block forms the mean itself (records_kernel<., FUSED>)
    if (pl.fused_pre && B < 64) nparts = (Nt + 511) / 512;   // ... and a few series: spread the fp64 record work over more blocks
    pl.nparts = (int)nparts;
    pl.part_chunk = (Nt + nparts - 1) / nparts;
    pl.nparts = (int)((Nt + pl.part_chunk - 1) / pl.part_chunk);
    pl.launches = 4;
    return pl;
}

// ---- workspace layouts (byte offsets into the handle's buffer)
constexpr int64_t REFINE_INPLACE_MAX_NT = 16384;        // lsp_periodogram_static: finish_kernel redoes its ill-conditioned frequencies itself up to this length
constexpr int64_t REFINE_LIST_MIN_NT = 2048;            // handle paths: longer series list them for refine_kernel (lsp_refine.cuh): flagged bins come in runs
                                                        // (low f, every alias of a nightly cadence) that one finish block would redo one after the other (C2: +21 us)
constexpr int64_t SHARED_E_BUDGET_DEFAULT = (int64_t)256 << 20;   // bytes of workspace the E tiles of the shared-time GEMM may take (per band)

struct SharedLayout {
    int64_t nsplit, gps, ng, nmb, nfb, x_row, band_nfb;
    bool fuse;
    size_t recB, xa, eb, wsv, wsx, vc, vcf, psum, pvar, peak, cnt, total;
};

// Shared-time batch: false if the sizes do not fit the kernel's grid.
bool shared_layout(const Plan& pl, int64_t B, int64_t Nt, int64_t Nf, int64_t e_budget, SharedLayout& L)
{
    int64_t nsplit = (Nt + SG_MAX_SPLIT - 1) / SG_MAX_SPLIT;
    int64_t gps = ((Nt + nsplit - 1) / nsplit + SG_KS - 1) / SG_KS;
    gps = (gps + SG_KPS - 1) / SG_KPS * SG_KPS;           // k-step groups per split: whole stages
    nsplit = (Nt + gps * SG_KS - 1) / (gps * SG_KS);
    L.nsplit = nsplit; L.gps = gps; L.ng = nsplit * gps;
    L.nmb = (B + SG_M - 1) / SG_M; L.nfb = (Nf + SG_F - 1) / SG_F;
    L.x_row = (Nf + 3) / 4 * 4;
    if (L.nmb * L.nfb * nsplit > 2147483647LL || L.ng > 65535 || nsplit > 65535) return false;
    L.fuse = (nsplit == 1);                               // one split: the GEMM's accumulators are the sums; steps 6-7 run in its epilogue
    size_t off = 0;
    L.recB = off; off = align_up(off + (size_t)Nt * sizeof(ulonglong2), 256);   // phases of the one time vector
    L.xa = off;   off = align_up(off + (size_t)L.nmb * L.ng * SG_A_GROUP, 256);
    // E = 8 bytes per (sample, frequency): made and consumed one band of frequency blocks at a time, so it takes O(Nt * band), not O(Nt * Nf)
    int64_t band = (e_budget > 0 ? e_budget : SHARED_E_BUDGET_DEFAULT) / (L.ng * (int64_t)SG_B_GROUP);
    const int64_t fill = (2 * 148 + L.nmb * nsplit - 1) / (L.nmb * nsplit);      // a band launch should still fill the device (two CTAs per SM)
    if (band < fill) band = fill;
    if (band > L.nfb) band = L.nfb;
    if (band < 1) band = 1;
    L.band_nfb = band;
    L.eb = off;   off = align_up(off + (size_t)band * L.ng * SG_B_GROUP, 256);
    L.wsv = off;  off = align_up(off + (size_t)nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    L.wsx = off;  if (!L.fuse) off = align_up(off + (size_t)B * nsplit * 2 * (size_t)L.x_row * sizeof(float), 256);
    L.vc = off;   off = align_up(off + (size_t)4 * (size_t)Nf * sizeof(double), 256);
    L.vcf = off;  off = align_up(off + (size_t)Nf * sizeof(float4), 256);
    L.psum = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    L.pvar = off; off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    L.peak = off; off = align_up(off + (size_t)B * sizeof(u64), 256);
    L.cnt = off;  off = align_up(off + (size_t)B * sizeof(unsigned), 256);
    L.total = off;
    return true;
}

struct Layout {
    size_t recA, recB, ws, ws1, recA1, psum, pvar, pw, peak, cnt, tab, total;
    int64_t tab_groups;          // k-step groups of one series' table (one chunk + padding); 0: no table
    size_t tab_bytes;
};

Layout device_layout(const Plan& pl, int64_t B, int64_t Nt, int64_t Nf, int64_t tab_series, bool gls)
{
    Layout L;
    const size_t n_samp = (size_t)B * (size_t)Nt;
    size_t off = 0;
    L.recA = off;  off = align_up(off + n_samp * sizeof(float4), 256);
    L.recB = off;  off = align_up(off + n_samp * sizeof(ulonglong2), 256);
    L.ws = off;    off = align_up(off + (size_t)B * pl.nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    L.ws1 = off;   if (gls) off = align_up(off + (size_t)B * pl.nsplit * 4 * (size_t)Nf * sizeof(float), 256);
    L.recA1 = off; if (gls) off = align_up(off + n_samp * sizeof(float4), 256);
    L.psum = off;  off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    L.pvar = off;  off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);
    L.pw = off;    if (gls) off = align_up(off + (size_t)B * pl.nparts * sizeof(double), 256);   // weighted form: sum of weights per block
    L.peak = off;  off = align_up(off + (size_t)B * sizeof(u64), 256);
    L.cnt = off;   off = align_up(off + (size_t)B * sizeof(unsigned), 256);
    L.tab_groups = 0; L.tab_bytes = 0; L.tab = off;
    if (pl.pipe == PLAN_PIPE_TENSOR && pl.L >= 128) {     // CTA-pair form: the fine-operand table of ONE time chunk (lsp_accum_umma_pair2.cuh)
        L.tab_groups = (pl.chunk_len + UM_KS - 1) / UM_KS + U2_TABLE_PAD_KSTEPS;
        L.tab_bytes = (size_t)tab_series * (size_t)L.tab_groups * U2_TABLE_BYTES_PER_KSTEP;
        off = align_up(off + L.tab_bytes, 256);
    }
    L.total = off;
    return L;
}

// steps 6-7: on short grids with several time splits the sum over them is spread over 8 threads per frequency
// Launch `kernel` as a programmatic dependent of the work before it in the stream (PDL): its CTAs may be scheduled while the
// predecessor drains; the kernel calls pdl_wait() before reading what the predecessor wrote.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

void launch_finish(const FinishParams& fp, int64_t B, cudaStream_t st, bool pdl = false)
{
    // blocks per series: all the frequency chunks of a single series; for a batch about four waves of blocks in all (each block
    // then loops over several chunks of its series)
    constexpr int64_t TARGET_BLOCKS = 4 * 8 * 148;
    const int64_t per_series = (TARGET_BLOCKS + B - 1) / B;
    if (fp.nsplit >= 4 && fp.Nf <= 65536) {               // (long grids have enough frequencies to fill the machine one thread each: 170 vs 360 us at C5)
        const int64_t nchunk = (fp.Nf + FIN_THREADS / 8 - 1) / (FIN_THREADS / 8);
        if (per_series < nchunk) launch_pdl(finish_kernel<8, true>, dim3((unsigned)per_series, (unsigned)B), dim3(FIN_THREADS), 0, st, pdl, fp);
        else launch_pdl(finish_kernel<8, false>, dim3((unsigned)nchunk, (unsigned)B), dim3(FIN_THREADS), 0, st, pdl, fp);
    } else {
        const int64_t nchunk = (fp.Nf + FIN_THREADS - 1) / FIN_THREADS;
        if (per_series < nchunk) launch_pdl(finish_kernel<1, true>, dim3((unsigned)per_series, (unsigned)B), dim3(FIN_THREADS), 0, st, pdl, fp);
        else launch_pdl(finish_kernel<1, false>, dim3((unsigned)nchunk, (unsigned)B), dim3(FIN_THREADS), 0, st, pdl, fp);
    }
}

// The list the fused epilogues append their ill-conditioned frequencies to (allocated on first use; its head is 0 between calls:
// refine_kernel clears it).
int refine_list(lsp_ctx* h, RefineList& L)
{
    constexpr size_t HEAD = 256, DONE = (size_t)REFINE_SPLIT_ENTRIES * sizeof(unsigned);
    constexpr size_t PARTIAL = (size_t)REFINE_SPLIT_ENTRIES * REFINE_MAX_SPLIT * 4 * sizeof(double);
    if (!h->refine_buf) {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, HEAD + DONE + PARTIAL + (size_t)REFINE_LIST_CAP * sizeof(int2));
        if (e != cudaSuccess) { h->last_cuda = (int)e; cudaGetLastError(); return LSP_ENOMEM; }
        e = cudaMemset(p, 0, HEAD + DONE);
        if (e != cudaSuccess) { cudaFree(p); return cuda_fail(h, e); }
        h->refine_buf = p;
    }
    char* base = static_cast<char*>(h->refine_buf);
    L.head = reinterpret_cast<unsigned*>(base);
    L.entry_done = reinterpret_cast<unsigned*>(base + HEAD);
    L.partial = reinterpret_cast<double*>(base + HEAD + DONE);
    L.items = reinterpret_cast<int2*>(base + HEAD + DONE + PARTIAL);
    return LSP_OK;
}

// After a fused epilogue: steps 6-7 again for the frequencies it listed (none on most grids: the kernel then returns at once).
cudaError_t launch_refine(const RefineList& list, const RefineSrc& src, const double* pvar, int nparts, float* P, int64_t p_stride,
                          int32_t* peak_idx, float* peak_val, u64* peak64, cudaStream_t st, bool gls = false,
                          const double* psum = nullptr, const double* pw = nullptr)
{
    RefineParams rp;
    rp.src = src; rp.list = list; rp.part_var = pvar; rp.nparts = nparts; rp.P = P; rp.p_stride = p_stride;
    rp.peak_idx = peak_idx; rp.peak_val = peak_val; rp.peak64 = peak64; rp.gls = gls ? 1 : 0;
    rp.part_sum = psum; rp.part_w = pw;
    // a programmatic dependent of the kernel before it (it waits before reading the list): its launch overlaps that kernel's tail
    return launch_pdl(refine_kernel, dim3(2 * 148), dim3(REFINE_THREADS), 0, st, true, rp);
}

bool use_shared_path(const lsp_ctx* h, int64_t t_stride, int64_t B, int64_t Nt, bool gls)
{
    return t_stride == 0 && B > 1 && !gls && h->opt_shared != 1 && h->opt_pipe == 0 &&
           (h->opt_shared == 2 || (B >= 16 && Nt >= 512));
}

// Shared-time batch (t_stride = 0): XC, XS as one dense GEMM over all series, CC, CS once per frequency (lsp_shared_gemm.cuh).
int run_device_shared(lsp_ctx* h, const double* t, const float* x, int64_t x_stride,
                      int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                      float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, cudaStream_t st)
{
    Plan pl = make_plan(h, B, Nt, Nf, 1);                 // pre-pass partition only
    SharedLayout L;
    if (!shared_layout(pl, B, Nt, Nf, h->opt_table_mb << 20, L)) return LSP_EINVAL;
    const int64_t nsplit = L.nsplit, gps = L.gps, ng = L.ng, nmb = L.nmb, nfb = L.nfb, x_row = L.x_row;
    const int64_t nbands = (nfb + L.band_nfb - 1) / L.band_nfb;
    const bool fuse = L.fuse;
    pl.pipe = PLAN_PIPE_TENSOR; pl.K = SG_F; pl.T = SG_THREADS; pl.nsplit = (int)nsplit; pl.nfb = (int)nfb; pl.L = 0;
    pl.split_len = gps * SG_KS; pl.launches = 5 + 2 * (int)nbands; pl.nchunks = (int)nbands; pl.chunk_len = 0;
    pl.kernel_name = fuse ? "shared_gemm_kernel<tcgen05.m128n256.f16+e5m2corr,TMA-fed,shared-times,fused-finish>"
                          : "shared_gemm_kernel<tcgen05.m128n256.f16+e5m2corr,TMA-fed,shared-times>";

    int rc = ensure(h, &h->buf, &h->buf_bytes, L.total);
    if (rc != LSP_OK) return rc;
    char* base = static_cast<char*>(h->buf);
    ulonglong2* recB = reinterpret_cast<ulonglong2*>(base + L.recB);
    float4* recA = reinterpret_cast<float4*>(base + L.recB);          // (no per-sample measurement records on this path: never written)
    unsigned char* xa = reinterpret_cast<unsigned char*>(base + L.xa);
    unsigned char* eb = reinterpret_cast<unsigned char*>(base + L.eb);
    float* ws_v = reinterpret_cast<float*>(base + L.wsv);
    float* ws_x = reinterpret_cast<float*>(base + L.wsx);
    double* vconst = reinterpret_cast<double*>(base + L.vc);
    float4* vconst_f = reinterpret_cast<float4*>(base + L.vcf);
    double* psum = reinterpret_cast<double*>(base + L.psum);
    double* pvar = reinterpret_cast<double*>(base + L.pvar);
    u64* peak64 = reinterpret_cast<u64*>(base + L.peak);
    unsigned* counter = reinterpret_cast<unsigned*>(base + L.cnt);

    const bool timing = h->opt_timing != 0;
    const int slot = (int)(h->timed_calls % TIMING_RING);
    cudaEvent_t* ev = h->ev[slot];
    if (timing) {
        for (int i = 0; i < 5; ++i)
            if (!ev[i]) LSP_CUDA(h, cudaEventCreate(&ev[i]));
        h->ev_chunks[slot] = 0;
        LSP_CUDA(h, cudaEventRecord(ev[0], st));
    }
    // ill-conditioned frequencies (lsp_refine.cuh): V comes from a single fp16 pass here too
    RefineSrc src;
    src.t = t; src.t_stride = 0; src.x = x; src.x_stride = x_stride; src.w = nullptr; src.w_stride = 0; src.f_min = f_min; src.df = df; src.Nt = Nt;
    const bool refine = h->opt_refine == 0;
    const double amp = refine ? refine_amplification(true, Nt) : 0.0;
    const double refine_thr = 1.0 - 1.0 / (refine ? amp : 10.0);
    const double redo_thr = (refine && refine_thr < 0.5) ? refine_thr : 0.5;      // the epilogue looks closer (fp64, list) above this R / Nt
    RefineList rlist = {};
    if (fuse && refine) { rc = refine_list(h, rlist); if (rc != LSP_OK) return rc; pl.launches += 1; }
    // steps 1-2 (per series: mean, variance, X; the phase records of series 0 serve all)
    dim3 gpre((unsigned)pl.nparts, (unsigned)B);
    const bool fused_pre = pl.fused_pre;                   // short series: step 1's sum inside the records kernel
    const int TRIG = 0;
    if (!fused_pre) {
        moments_kernel<<<gpre, 256, 0, st>>>(x, x_stride, Nt, pl.part_chunk, psum, peak64, counter);
        LSP_CUDA(h, cudaGetLastError());
    } else pl.launches -= 1;
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[1], st));
    if (fused_pre) records_kernel<true, true><<<gpre, 256, 0, st>>>(t, 0, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter, origin_offset(f_min, df, Nf), TRIG);
    else records_kernel<true, false><<<gpre, 256, 0, st>>>(t, 0, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter, origin_offset(f_min, df, Nf), TRIG);
    LSP_CUDA(h, cudaGetLastError());
    // CC, CS once per frequency
    const bool pdl = h->opt_pdl != 1;                      // programmatic dependents: each kernel's launch overlaps its predecessor's tail
    LSP_CUDA(h, launch_pdl(shared_v_kernel, dim3((unsigned)((Nf + 7) / 8), (unsigned)nsplit), dim3(256), 0, st, pdl, (const ulonglong2*)recB, Nt, Nf, gps * SG_KS, ws_v));
    if (fuse) {
        LSP_CUDA(h, launch_pdl(shared_vconst_kernel, dim3((unsigned)((Nf + 255) / 256)), dim3(256), 0, st, pdl, (const float*)ws_v, (int)nsplit, Nf, Nt, vconst, vconst_f, redo_thr));
    }
    LSP_CUDA(h, launch_pdl(shared_x_kernel, dim3((unsigned)nmb, (unsigned)ng), dim3(256), 0, st, pdl, x, x_stride, (const double*)psum, (const double*)pvar, pl.nparts, B, Nt, xa, (int)ng));
    // step 3 for every (sample, frequency) once, and steps 4-5, the contraction: one band of frequency blocks at a time
    // (E tiles of the band -> GEMM over the band; the same buffer serves every band)
    SharedGemmParams gp;
    gp.xa = xa; gp.eb = eb; gp.ws_x = ws_x; gp.B = B; gp.Nf = Nf; gp.x_row = x_row;
    gp.nmb = (int)nmb; gp.nfb_total = (int)nfb; gp.nsplit = (int)nsplit; gp.ng = (int)ng; gp.groups_per_split = (int)gps;
    gp.vconst = fuse ? vconst : nullptr; gp.vconst_f = vconst_f; gp.part_var = pvar; gp.P = P; gp.p_stride = p_stride;
    gp.peak_idx = peak_idx; gp.peak_val = peak_val; gp.peak64 = peak64; gp.counter = counter; gp.Nt = Nt; gp.nparts = pl.nparts;
    gp.list = rlist; gp.refine_thr = refine_thr;
    const float refine_pow = refine ? refine_power(true, Nt, gps * SG_KS) : INFINITY;     // a time split is one accumulation window here
    LSP_CUDA(h, cudaFuncSetAttribute(shared_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SG_SMEM));
    for (int64_t band = 0; band < nbands; ++band) {
        const int64_t nb0 = band * L.band_nfb;
        const int64_t nb_n = (nfb - nb0 < L.band_nfb) ? nfb - nb0 : L.band_nfb;
        LSP_CUDA(h, launch_pdl(shared_e_kernel, dim3((unsigned)nb_n, (unsigned)ng), dim3(256), 0, st, pdl, (const ulonglong2*)recB, Nt, Nf, eb, (int)ng, (int)nb0));
        if (timing && band == 0) LSP_CUDA(h, cudaEventRecord(ev[2], st));
        gp.nb0 = (int)nb0; gp.nfb = (int)nb_n;
        LSP_CUDA(h, launch_pdl(shared_gemm_kernel, dim3((unsigned)(nmb * nb_n * nsplit)), dim3(SG_THREADS), SG_SMEM, st, pdl, gp));
    }
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[3], st));
    if (fuse) {                                           // steps 6-7 ran in the GEMM's epilogue
        if (refine) LSP_CUDA(h, launch_refine(rlist, src, pvar, pl.nparts, P, p_stride, peak_idx, peak_val, peak64, st));
        if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
        h->plan = pl;
        return LSP_OK;
    }
    // steps 6-7
    FinishParams fp;
    fp.ws = ws_v; fp.part_var = pvar; fp.P = P; fp.p_stride = p_stride;
    fp.peak_idx = peak_idx; fp.peak_val = peak_val; fp.peak64 = peak64; fp.counter = counter;
    fp.Nt = Nt; fp.Nf = Nf; fp.nsplit = (int)nsplit; fp.nparts = pl.nparts;
    fp.x_scaled = 1; fp.ws1 = nullptr; fp.ws_x = ws_x; fp.x_row = x_row;
    fp.src = src; fp.refine_amp = amp; fp.refine_pow = refine_pow;
    fp.list = RefineList{};
    const bool listed = refine && Nt > REFINE_LIST_MIN_NT;
    if (listed) { rc = refine_list(h, fp.list); if (rc != LSP_OK) return rc; pl.launches += 1; }
    launch_finish(fp, B, st);
    LSP_CUDA(h, cudaGetLastError());
    if (listed) LSP_CUDA(h, launch_refine(fp.list, src, pvar, pl.nparts, P, p_stride, peak_idx, peak_val, peak64, st, false, psum));
    if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
    h->plan = pl;
    return LSP_OK;
}

// What the call will run (shared by run_device and lsp_reserve).
struct Route { Plan pl; bool tensor, small, duo, duo_fuse, pair, fuse_pre, gls_fused; int64_t tab_series; };

int route(const lsp_ctx* h, int64_t t_stride, int64_t B, int64_t Nt, int64_t Nf, bool gls, Route& r, bool weighted = false)
{
    r.tab_series = (t_stride == 0) ? 1 : B;
    // (per-sample weights: every form carries them; generalised periodogram on the FP32 form: one pass with K <= 20 frequencies per thread)
    r.pl = make_plan(h, B, Nt, Nf, r.tab_series, 0, gls ? GLS_FUSED_MAX_K : 32);
    Plan& pl = r.pl;
    if (pl.K == 0) return LSP_EINVAL;
    r.tensor = pl.pipe == PLAN_PIPE_TENSOR;
    r.pair = r.tensor && pl.L >= 128;                     // CTA pairs, table-fed (lsp_accum_umma_pair2.cuh)
    r.small = r.tensor && !r.pair;                        // 128 x L frequencies per CTA, two or three CTAs per SM
    r.duo = r.small && pl.L == 16 && B >= 2;              // batches: two series per CTA (lsp_accum_umma_duo.cuh)
    // one CTA sees all samples of its series in one drain window: steps 6-7 run in its epilogue, no workspace round trip
    r.duo_fuse = r.duo && !gls && pl.nsplit == 1 && Nt <= (h->opt_flush ? h->opt_flush : 2048);
    r.gls_fused = false;
    if (!r.tensor) {
        const KernelEntry* ke = find_kernel(pl.K);
        if (!ke || pl.T < 32 || pl.T > ke->max_t || (pl.T % 32) != 0) return LSP_EINVAL;
        pl.kernel_name = weighted ? ke->name_weighted : ke->name;
        r.gls_fused = gls && ke->fn_gls != nullptr;          // (a forced K > 20 takes the two-pass route)
        if (r.gls_fused) pl.kernel_name = weighted ? ke->name_gls_weighted : ke->name_gls;
    } else if (r.pair) {
        if (h->opt_corr) pl.kernel_name = weighted ? "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16,hi+lo,fine-table,weighted>"
                                                   : "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16,hi+lo,fine-table>";
        else
        pl.kernel_name = weighted ? "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16+e5m2corr,fine-table,weighted>"
                                  : "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16+e5m2corr,fine-table>";
        pl.launches = 3 + 2 * pl.nchunks;
    } else if (r.duo) {
        pl.kernel_name = r.duo_fuse ? "accum_umma_duo_kernel<tcgen05.m128n128k16.f16,hi+lo,2 series x 64 x 32,fused-finish>"
                       : (weighted ? "accum_umma_duo_kernel<tcgen05.m128n128k16.f16,hi+lo,2 series x 64 x 32,weighted>"
                                   : "accum_umma_duo_kernel<tcgen05.m128n128k16.f16,hi+lo,2 series x 64 x 32>");
        if (r.duo_fuse) pl.launches = 3;
    } else {
        if (weighted)
        pl.kernel_name = pl.L == 16 ? "accum_umma_small_kernel<tcgen05.m128n32k16.f16,hi+lo,weighted>"
                       : (pl.L == 32 ? "accum_umma_small_kernel<tcgen05.m128n64k16.f16,hi+lo,weighted>"
                                     : "accum_umma_small_kernel<tcgen05.m128n128k16.f16,hi+lo,weighted>");
        else
        pl.kernel_name = pl.L == 16 ? "accum_umma_small_kernel<tcgen05.m128n32k16.f16,hi+lo>"
                       : (pl.L == 32 ? "accum_umma_small_kernel<tcgen05.m128n64k16.f16,hi+lo>"
                                     : "accum_umma_small_kernel<tcgen05.m128n128k16.f16,hi+lo>");
    }
    // short grids, short series: steps 1-2 inside the accumulate kernel (accum_umma_small_kernel<..., FUSED_PRE>): two launches per call
    r.fuse_pre = r.small && !r.duo && !gls && !weighted && Nt <= 16384 && h->opt_pdl != 1;
    if (r.fuse_pre) { pl.launches = 2; pl.nparts = 1; pl.part_chunk = Nt; pl.fused_pre = false; }
    // ... and of the batch kernel (accum_umma_duo_kernel<FUSED_PRE>); with the fused epilogue only where one CTA owns the whole series
    // (the CTA that resets the arg-max cell is then the only one that updates it)
    if (r.duo && !gls && !weighted && Nt <= 16384 && h->opt_pdl != 1 && (!r.duo_fuse || pl.nfb == 1)) {
        r.fuse_pre = true;
        pl.launches = r.duo_fuse ? 1 : 2; pl.nparts = 1; pl.part_chunk = Nt; pl.fused_pre = false;
    }
    if (gls && !r.gls_fused) pl.launches += 1 + (r.pair ? pl.nchunks : 1);   // unit records + second accumulate pass
    const int64_t units = (r.duo ? (B + 1) / 2 : B) * (int64_t)pl.nsplit * pl.nfb;
    if (units > 2147483647LL) return LSP_EINVAL;
    return LSP_OK;
}

int run_device(lsp_ctx* h,
               const double* t, int64_t t_stride, const float* x, int64_t x_stride,
               int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
               float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, cudaStream_t st, bool gls = false,
               const float* w = nullptr, int64_t w_stride = 0)
{
    const bool weighted = w != nullptr;                    // weighted generalised periodogram (implies gls)
    if (use_shared_path(h, t_stride, B, Nt, gls))
        return run_device_shared(h, t, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride, peak_idx, peak_val, st);
    Route r;
    int rc = route(h, t_stride, B, Nt, Nf, gls, r, weighted);
    if (rc != LSP_OK) return rc;
    Plan& pl = r.pl;
    const bool tensor = r.tensor;                          // tensor-core forms: X scaled to unit variance
    const KernelEntry* ke = tensor ? nullptr : find_kernel(pl.K);

    const Layout L = device_layout(pl, B, Nt, Nf, r.tab_series, gls);
    rc = ensure(h, &h->buf, &h->buf_bytes, L.total);
    if (rc != LSP_OK) return rc;
    const size_t n_samp = (size_t)B * (size_t)Nt;
    char* base = static_cast<char*>(h->buf);
    float4* recA = reinterpret_cast<float4*>(base + L.recA);
    ulonglong2* recB = reinterpret_cast<ulonglong2*>(base + L.recB);
    float* ws = reinterpret_cast<float*>(base + L.ws);
    float* ws1 = gls ? reinterpret_cast<float*>(base + L.ws1) : nullptr;          // unit-weight pass: sum cos, sum sin
    float4* recA1 = gls ? reinterpret_cast<float4*>(base + L.recA1) : nullptr;
    double* psum = reinterpret_cast<double*>(base + L.psum);
    double* pvar = reinterpret_cast<double*>(base + L.pvar);
    double* pw = reinterpret_cast<double*>(base + L.pw);
    u64* peak64 = reinterpret_cast<u64*>(base + L.peak);
    unsigned* counter = reinterpret_cast<unsigned*>(base + L.cnt);
    unsigned char* table = reinterpret_cast<unsigned char*>(base + L.tab);

    const bool timing = h->opt_timing != 0;
    const int slot = (int)(h->timed_calls % TIMING_RING);
    cudaEvent_t* ev = h->ev[slot];
    cudaEvent_t* evc = h->evc[slot];
    const bool chunk_timing = timing && r.pair && pl.nchunks > 1 && pl.nchunks <= TIMING_MAX_CHUNKS;
    if (timing) {
        for (int i = 0; i < 5; ++i)
            if (!ev[i]) LSP_CUDA(h, cudaEventCreate(&ev[i]));
        if (chunk_timing)
            for (int i = 0; i < 2 * pl.nchunks; ++i)
                if (!evc[i]) LSP_CUDA(h, cudaEventCreate(&evc[i]));
        h->ev_chunks[slot] = chunk_timing ? pl.nchunks : 0;
        LSP_CUDA(h, cudaEventRecord(ev[0], st));
    }

    // steps 1-2
    dim3 gpre((unsigned)pl.nparts, (unsigned)B);
    const bool fused_pre = pl.fused_pre && !weighted;      // short series: step 1's sum inside the records kernel
    const int TRIG = tensor ? 0 : 1;                       // (cos d_j, sin d_j) of the FP32-pipe form's recurrence
    const int64_t order_stride = (tensor && h->opt_order != 1) ? record_order_stride(Nt) : 1;   // tensor forms: samples in a golden-ratio stride order (lsp_prepass.cuh)
    if (r.fuse_pre) {                                     // (done by the accumulate kernel itself)
        if (timing) LSP_CUDA(h, cudaEventRecord(ev[1], st));
    } else {
    if (!fused_pre) {
        moments_kernel<<<gpre, 256, 0, st>>>(x, x_stride, Nt, pl.part_chunk, psum, peak64, counter, w, w_stride, pw);
        LSP_CUDA(h, cudaGetLastError());
    } else pl.launches -= 1;
    if (timing) LSP_CUDA(h, cudaEventRecord(ev[1], st));
    if (weighted) records_weighted_kernel<<<gpre, 256, 0, st>>>(t, t_stride, x, x_stride, w, w_stride, Nt, pl.part_chunk, f_min, df, psum, pw, recA, recA1, recB, pvar, origin_offset(f_min, df, Nf), TRIG, order_stride);
    else if (fused_pre) records_kernel<false, true><<<gpre, 256, 0, st>>>(t, t_stride, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter, origin_offset(f_min, df, Nf), TRIG, order_stride);
    else records_kernel<false, false><<<gpre, 256, 0, st>>>(t, t_stride, x, x_stride, Nt, pl.part_chunk, f_min, df, psum, recA, recB, pvar, peak64, counter, origin_offset(f_min, df, Nf), TRIG, order_stride);
    LSP_CUDA(h, cudaGetLastError());
    }
    if (weighted && !r.gls_fused) pl.launches -= 1;       // (the weight records were written by records_weighted_kernel)
    if (gls && !weighted && !r.gls_fused) {
        unit_records_kernel<<<(unsigned)((n_samp + 255) / 256), 256, 0, st>>>(recA, recA1, (int64_t)n_samp);
        LSP_CUDA(h, cudaGetLastError());
    }

    RefineSrc src;                                        // the raw series, for the frequencies whose sums are ill-conditioned
    src.t = t; src.t_stride = t_stride; src.x = x; src.x_stride = x_stride; src.w = w; src.w_stride = w_stride; src.f_min = f_min; src.df = df; src.Nt = Nt;
    const bool refine = h->opt_refine == 0;
    RefineList rlist = {};
    if (r.duo_fuse && refine) { rc = refine_list(h, rlist); if (rc != LSP_OK) return rc; pl.launches += 1; }

    // steps 3-5 (generalised periodogram: a second pass with unit weights gives sum cos, sum sin in ws1)
    const int npass = (gls && !r.gls_fused) ? 2 : 1;
    // short grids, one pass: records -> accumulate -> finish as programmatic dependents (launch latency and CTA set-up overlap the predecessor's tail)
    const bool pdl_small = r.small && !r.duo && !gls && h->opt_pdl != 1;
    // drain interval of D_W and D_V: 2,048 samples; 4,096 in the CTA-pair form, where a drain stalls the whole pipeline of the pair
    // (2,048 / 4,096 / 8,192: 21.6 / 20.5 / 20.2 ms at C5).  The expected truncation loss of a D_W window is added back at its drain
    // (tc_trunc_comp); on series with a trend the model is only approximate and the residual grows with the window
    const int64_t flush_default = r.pair ? 4096 : 2048;
    const int flush_ksteps = (int)(((h->opt_flush ? h->opt_flush : flush_default) + UM_KS - 1) / UM_KS);
    // strong lines on the tensor forms are refined as well (refine_power, lsp_refine.cuh); the window is the drain window or the time split
    const int64_t window = ((int64_t)flush_ksteps * UM_KS < pl.split_len) ? (int64_t)flush_ksteps * UM_KS : pl.split_len;
    const float refine_pow = refine ? refine_power(tensor, Nt, window) : INFINITY;
    if (r.pair) {
        // CTA-pair form, one time chunk at a time: table pre-pass, then the accumulate launch(es) that read it
        const int64_t half_stride = L.tab_groups * (int64_t)UP_GROUP_BYTES;
        const int64_t series_stride = L.tab_groups * (int64_t)U2_TABLE_BYTES_PER_KSTEP;
        void (*pair_kernel)(const UmmaPairParams) = h->opt_corr ? accum_umma_pair2_kernel<true> : accum_umma_pair2_kernel<false>;
        LSP_CUDA(h, cudaFuncSetAttribute(pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)U2_SMEM));
        for (int c = 0; c < pl.nchunks; ++c) {
            const int64_t j0 = (int64_t)c * pl.chunk_len;
            const int64_t len = (Nt - j0 < pl.chunk_len) ? Nt - j0 : pl.chunk_len;
            const int64_t groups = (len + UM_KS - 1) / UM_KS + U2_TABLE_PAD_KSTEPS;
            umma_ftable_pair_kernel<<<dim3((unsigned)groups, (unsigned)r.tab_series), 512, 0, st>>>(recB, j0, j0 + len, Nt, table, half_stride, series_stride, (int)h->opt_corr);
            LSP_CUDA(h, cudaGetLastError());
            if (timing && c == 0) LSP_CUDA(h, cudaEventRecord(ev[2], st));
            if (chunk_timing) LSP_CUDA(h, cudaEventRecord(evc[2 * c], st));
            const int nsplit_c = (int)((len + pl.split_len - 1) / pl.split_len);
            for (int pass = 0; pass < npass; ++pass) {
                UmmaPairParams pp;
                UmmaParams& up = pp.u;
                up.recA = pass ? recA1 : recA; up.recB = recB; up.recW = nullptr; up.part_var = pvar; up.ws = pass ? ws1 : ws; up.Nt = Nt; up.Nf = Nf;
                up.split_len = pl.split_len; up.nsplit = pl.nsplit; up.nfb = pl.nfb; up.nparts = pl.nparts;
                up.flush_ksteps = flush_ksteps;
                up.trunc_ulps = h->opt_trunc == 0 ? -1.f : (h->opt_trunc == 1 ? 0.f : 1e-3f * (float)h->opt_trunc);
                up.unit_x = pass;
                pp.btable = table; pp.half_stride = half_stride; pp.table_stride = (r.tab_series == 1) ? 0 : series_stride;
                pp.j0 = j0; pp.chunk_len = len; pp.accumulate = c > 0 ? 1 : 0;
                pp.recW = weighted ? recA1 : nullptr;
                pp.nsplit_grid = nsplit_c;                  // only the splits this chunk has; pl.nsplit still strides `ws`
                const int64_t units = B * (int64_t)nsplit_c * pl.nfb;
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3((unsigned)units); cfg.blockDim = dim3(U2_THREADS); cfg.dynamicSmemBytes = U2_SMEM; cfg.stream = st;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                LSP_CUDA(h, cudaLaunchKernelEx(&cfg, pair_kernel, pp));
            }
            if (chunk_timing) LSP_CUDA(h, cudaEventRecord(evc[2 * c + 1], st));
        }
    } else {
        if (timing) LSP_CUDA(h, cudaEventRecord(ev[2], st));
        const int64_t units = (r.duo ? (B + 1) / 2 : B) * (int64_t)pl.nsplit * pl.nfb;
        for (int pass = 0; pass < npass; ++pass) {
            const float4* rA = pass ? recA1 : recA;
            float* wsp = pass ? ws1 : ws;
            if (tensor) {
                UmmaParams up;
                up.recA = rA; up.recB = recB; up.recW = weighted ? recA1 : nullptr; up.part_var = pvar; up.ws = wsp; up.Nt = Nt; up.Nf = Nf;
                up.split_len = pl.split_len; up.nsplit = pl.nsplit; up.nfb = pl.nfb; up.nparts = pl.nparts;
                up.flush_ksteps = flush_ksteps; up.trunc_ulps = h->opt_trunc == 1 ? 0.f : -1.f; up.unit_x = pass;   // (the model, or none: LSP_PARAM_TRUNC = 1)
                up.t = t; up.t_stride = t_stride; up.x = x; up.x_stride = x_stride; up.f_min = f_min; up.df = df;
                up.part_var_out = pvar; up.part_sum_out = psum; up.peak64 = peak64; up.counter = counter;
                if (r.duo) {
                    UmmaDuoParams dp;
                    dp.u = up; dp.B = B;
                    dp.fuse = r.duo_fuse ? 1 : 0; dp.P = P; dp.p_stride = p_stride;
                    dp.peak_idx = peak_idx; dp.peak_val = peak_val; dp.peak64 = peak64; dp.counter = counter;
                    dp.list = rlist;
                    dp.refine_r2 = INFINITY;
                    if (rlist.head) { const double thr = (1.0 - 1.0 / refine_amplification(true, Nt)) * (double)Nt; dp.refine_r2 = (float)(thr * thr); }
                    void (*duo_kernel)(const UmmaDuoParams) = weighted ? accum_umma_duo_kernel<false, true>
                                                            : (r.fuse_pre ? accum_umma_duo_kernel<true> : accum_umma_duo_kernel<false>);
                    LSP_CUDA(h, cudaFuncSetAttribute(duo_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UD_SMEM));
                    duo_kernel<<<(unsigned)units, US_THREADS, UD_SMEM, st>>>(dp);
                } else {
#define LSP_LAUNCH_SMALL(LL, NS, MINB) do { \
                    if (weighted) { \
                    LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_small_kernel<LL, NS, MINB, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UmmaSmall<LL, NS>::SMEM)); \
                    accum_umma_small_kernel<LL, NS, MINB, false, true><<<(unsigned)units, US_THREADS, UmmaSmall<LL, NS>::SMEM, st>>>(up); \
                    LSP_CUDA(h, cudaGetLastError()); } else \
                    if (r.fuse_pre) { \
                    LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_small_kernel<LL, NS, MINB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UmmaSmall<LL, NS>::SMEM)); \
                    accum_umma_small_kernel<LL, NS, MINB, true><<<(unsigned)units, US_THREADS, UmmaSmall<LL, NS>::SMEM, st>>>(up); \
                    LSP_CUDA(h, cudaGetLastError()); } else { \
                    LSP_CUDA(h, cudaFuncSetAttribute(accum_umma_small_kernel<LL, NS, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)UmmaSmall<LL, NS>::SMEM)); \
                    LSP_CUDA(h, launch_pdl(accum_umma_small_kernel<LL, NS, MINB>, dim3((unsigned)units), dim3(US_THREADS), UmmaSmall<LL, NS>::SMEM, st, pdl_small, up)); } } while (0)
                    if (pl.L == 16) LSP_LAUNCH_SMALL(16, 4, 3);
                    else if (pl.L == 32) LSP_LAUNCH_SMALL(32, 4, 2);
                    else if (pl.L == 64) LSP_LAUNCH_SMALL(64, 4, 2);
                    else return LSP_EINVAL;
#undef LSP_LAUNCH_SMALL
                }
            } else {
                AccumParams ap;
                ap.recW = weighted ? recA1 : nullptr;
                ap.recA = rA; ap.recB = recB; ap.ws = wsp; ap.ws1 = ws1; ap.Nt = Nt; ap.Nf = Nf;
                ap.split_len = pl.split_len; ap.nsplit = pl.nsplit; ap.nfb = pl.nfb; ap.flush_tiles = pl.flush_tiles;
                // the whole split inside one fold interval: the register partials go straight to `ws` (no shared-memory accumulators)
                const bool direct = !weighted && pl.split_len <= (int64_t)pl.flush_tiles * TILE_Z;
                const size_t smem = accum_smem_bytes(ke, pl.T, weighted, direct, r.gls_fused);
                const accum_fn fn = r.gls_fused ? (weighted ? ke->fn_gls_weighted : (direct ? ke->fn_gls_direct : ke->fn_gls))
                                                : (weighted ? ke->fn_weighted : (direct ? ke->fn_direct : ke->fn));
                LSP_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                fn<<<(unsigned)units, pl.T, smem, st>>>(ap);
            }
            LSP_CUDA(h, cudaGetLastError());
        }
    }
    LSP_CUDA(h, cudaGetLastError());

    if (timing) LSP_CUDA(h, cudaEventRecord(ev[3], st));

    if (r.duo_fuse) {
        if (refine) LSP_CUDA(h, launch_refine(rlist, src, pvar, pl.nparts, P, p_stride, peak_idx, peak_val, peak64, st));
        if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }
        h->plan = pl;
        return LSP_OK;
    }
    // steps 6-7
    FinishParams fp;
    fp.ws = ws; fp.part_var = pvar; fp.P = P; fp.p_stride = p_stride;
    fp.peak_idx = peak_idx; fp.peak_val = peak_val; fp.peak64 = peak64; fp.counter = counter;
    fp.Nt = Nt; fp.Nf = Nf; fp.nsplit = pl.nsplit; fp.nparts = pl.nparts;
    fp.x_scaled = tensor ? 1 : 0;
    fp.ws1 = ws1;
    fp.ws_x = nullptr; fp.x_row = 0;
    fp.src = src; fp.refine_amp = refine ? refine_amplification(tensor, Nt, gls, r.pair) : 0.0;
    fp.refine_pow = refine_pow;
    fp.list = RefineList{};
    // generalised form: its flagged frequencies come in runs (every alias of a nightly cadence), which one finish block would redo one
    // after the other: always through the list, a block or warp per frequency (C2-shaped call: steps 6-7 0.053 -> 0.02 ms)
    const bool listed = refine && (Nt > REFINE_LIST_MIN_NT || gls);
    if (listed) { rc = refine_list(h, fp.list); if (rc != LSP_OK) return rc; pl.launches += 1; }
    launch_finish(fp, B, st, pdl_small);
    LSP_CUDA(h, cudaGetLastError());
    if (listed) LSP_CUDA(h, launch_refine(fp.list, src, pvar, pl.nparts, P, p_stride, peak_idx, peak_val, peak64, st, gls, psum, weighted ? pw : nullptr));
    if (timing) { LSP_CUDA(h, cudaEventRecord(ev[4], st)); h->timed_calls++; }

    h->plan = pl;
    return LSP_OK;
}

// Host-buffer batches: into how many chunks of series (1, 2 or HOST_PIPE_CHUNKS) the call is cut so that the copies of one chunk
// overlap the compute of its neighbours.  A coarse model decides: copies at ~50 GB/s each way; compute from the terms and the rate
// of the form the plan picks, times the wave quantisation a smaller grid suffers (a chunk of an FP32-form batch that is 1.15 waves
// long costs two); chunks are taken only where the modelled pipelined time beats the serial one by >= 10 %.
int host_pipe_chunks(const lsp_ctx* h, bool share_t, int64_t B, int64_t Nt, int64_t Nf, bool want_P)
{
    const double t_in = ((double)(share_t ? 1 : B) * Nt * 8.0 + (double)B * Nt * 4.0) / 50e9;
    const double t_out = (want_P ? (double)B * Nf * 4.0 : 0.0) / 50e9;
    if (B < 64 || t_in + t_out < 150e-6) return 1;
    const double terms = (double)B * (double)Nt * (double)Nf;
    bool fp32_form = false;
    auto grid = [&](int64_t nb, double& units, double& slots, double& rate) {
        if (use_shared_path(h, share_t ? 0 : Nt, nb, Nt, false)) {
            units = (double)((nb + SG_M - 1) / SG_M) * (double)((Nf + SG_F - 1) / SG_F); slots = 2.0 * h->sm_count; rate = 5e13;
            return true;
        }
        Route r;
        if (route(h, share_t ? 0 : Nt, nb, Nt, Nf, false, r) != LSP_OK) return false;
        units = (double)(r.duo ? (nb + 1) / 2 : nb) * r.pl.nsplit * r.pl.nfb;
        if (r.tensor) { slots = (double)(r.duo ? 2 : plan_umma_ctas_per_sm(r.pl.L)) * h->sm_count; rate = r.pair ? 5e13 : 1.2e13; }
        else { slots = (double)plan_ctas_per_sm(r.pl.K, r.pl.T, r.pl.split_len <= PLAN_FOLD_SAMPLES) * h->sm_count; rate = 4.5e12; fp32_form = true; }
        return true;
    };
    double u1, s1, rate;
    if (!grid(B, u1, s1, rate)) return 1;
    const double t_comp = terms / rate;
    const double waves1 = u1 > s1 ? std::ceil(u1 / s1) : 1.0;
    const double serial = t_in + t_comp + t_out;
    int best = 1; double best_t = serial * 0.9;
    for (int n = 2; n <= HOST_PIPE_CHUNKS; n *= 2) {
        double un, sn, rn;
        if (!grid((B + n - 1) / n, un, sn, rn)) continue;
        const double wavesn = un > sn ? std::ceil(un / sn) : 1.0;
        // waves x work per CTA, relative to the whole batch in one call (a chunk of a tensor-form batch may be planned with more, shorter
        // CTAs: un != u1 / n; measured at C4: 4 chunks 1.40 ms, 2 chunks 1.61 ms).  FP32 form: every split pays its fixed cost again and the
        // finish step reads them all: a wave of a chunk is charged like a wave of the whole batch (C4S: 1 chunk 2.85 ms, 4 chunks 3.26 ms)
        const double rel = fp32_form ? (n * wavesn) / waves1 : (wavesn / un) / (waves1 / u1);
        const double comp = t_comp * rel * (u1 > s1 ? 1.0 : std::fmax(1.0, n * 0.35));   // under-filled grids: chunks do not get n times shorter
        const double pipe = std::fmax(t_in + (comp + t_out) / n, std::fmax(comp + (t_in + t_out) / n, t_out + (t_in + comp) / n));
        if (pipe < best_t) { best_t = pipe; best = n; }
    }
    return best;
}

bool bad_grid(double f_min, double df) {
    return !(std::isfinite(f_min) && std::isfinite(df)) || f_min < 0.0 || df < 0.0;
}

// Argument checks shared by the batched entry points (device and host forms).
int check_batch_args(lsp_ctx* h, const void* t, const void* x, int64_t B, int64_t Nt, int64_t min_nt,
                     double f_min, double df, int64_t Nf, const void* P, const void* peak_idx, const void* peak_val)
{
    if (!h || !t || !x) return LSP_EINVAL;
    if (B < 1 || B > 65535 || Nt < min_nt || Nf < 1 || Nt > 2000000000LL || Nf > 2000000000LL) return LSP_EINVAL;   // B: grid.y of the pre-pass / finish kernels
    if (bad_grid(f_min, df)) return LSP_EINVAL;
    if ((peak_idx == nullptr) != (peak_val == nullptr)) return LSP_EINVAL;
    if (!P && !peak_idx) return LSP_EINVAL;
    return LSP_OK;
}

int check_strides(int64_t t_stride, int64_t x_stride, int64_t p_stride, int64_t B, int64_t Nt, int64_t Nf, const void* P)
{
    if (B > 1) {
        if (t_stride != 0 && std::llabs(t_stride) < Nt) return LSP_EINVAL;
        if (std::llabs(x_stride) < Nt) return LSP_EINVAL;
        if (P && std::llabs(p_stride) < Nf) return LSP_EINVAL;
    }
    return LSP_OK;
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
    if (h->refine_buf) cudaFree(h->refine_buf);
    if (h->stage) cudaFree(h->stage);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    for (cudaEvent_t e : h->ev_pipe) if (e) cudaEventDestroy(e);
    for (int r = 0; r < TIMING_RING; ++r) {
        for (int i = 0; i < 5; ++i) if (h->ev[r][i]) cudaEventDestroy(h->ev[r][i]);
        for (int i = 0; i < 2 * TIMING_MAX_CHUNKS; ++i) if (h->evc[r][i]) cudaEventDestroy(h->evc[r][i]);
    }
    delete h;
    return LSP_OK;
}

int lsp_set_param(lsp_handle h, int key, int64_t value)
{
    if (!h || value < 0) return LSP_EINVAL;
    switch (key) {
        case LSP_PARAM_K:          if (value && !plan_valid_K((int)value)) return LSP_EINVAL; h->opt_K = value; break;
        case LSP_PARAM_THREADS:    if (value && (value < 32 || value > 256 || value % 32)) return LSP_EINVAL; h->opt_T = value; break;
        case LSP_PARAM_NSPLIT:     h->opt_nsplit = value; break;
        case LSP_PARAM_PIPE:       if (value > LSP_PIPE_TENSOR) return LSP_EINVAL; h->opt_pipe = value; break;
        case LSP_PARAM_FLUSH:      h->opt_flush = value; break;
        case LSP_PARAM_TIMING:     if (value > 1) return LSP_EINVAL; h->opt_timing = value; break;
        case LSP_PARAM_TABLE_MB:   if (value > (1 << 20)) return LSP_EINVAL; h->opt_table_mb = value; break;
        case LSP_PARAM_COARSE:     if (value && value != 16 && value != 32 && value != 64 && value != 128) return LSP_EINVAL; h->opt_coarse = value; break;
        case LSP_PARAM_TRUNC:      if (value > 4000) return LSP_EINVAL; h->opt_trunc = value; break;
        case LSP_PARAM_ORDER:      if (value > 1) return LSP_EINVAL; h->opt_order = value; break;
        case LSP_PARAM_SHARED:     if (value > 2) return LSP_EINVAL; h->opt_shared = value; break;
        case LSP_PARAM_PDL:        if (value > 1) return LSP_EINVAL; h->opt_pdl = value; break;
        case LSP_PARAM_CORR:       if (value > 1) return LSP_EINVAL; h->opt_corr = value; break;
        case LSP_PARAM_REFINE:     if (value > 1) return LSP_EINVAL; h->opt_refine = value; break;
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
        case LSP_PARAM_PIPE:       *value = h->opt_pipe; break;
        case LSP_PARAM_FLUSH:      *value = h->opt_flush; break;
        case LSP_PARAM_TIMING:     *value = h->opt_timing; break;
        case LSP_PARAM_TABLE_MB:   *value = h->opt_table_mb; break;
        case LSP_PARAM_COARSE:     *value = h->opt_coarse; break;
        case LSP_PARAM_TRUNC:      *value = h->opt_trunc; break;
        case LSP_PARAM_ORDER:      *value = h->opt_order; break;
        case LSP_PARAM_SHARED:     *value = h->opt_shared; break;
        case LSP_PARAM_PDL:        *value = h->opt_pdl; break;
        case LSP_PARAM_CORR:       *value = h->opt_corr; break;
        case LSP_PARAM_REFINE:     *value = h->opt_refine; break;
        default: return LSP_EINVAL;
    }
    return LSP_OK;
}

int lsp_reserve(lsp_handle h, int64_t B, int shared_t, int64_t Nt, int64_t Nf, int generalised)
{
    if (!h || B < 1 || B > 65535 || Nt < 2 || Nf < 1 || Nt > 2000000000LL || Nf > 2000000000LL) return LSP_EINVAL;
    DeviceGuard g(h->device);
    const int64_t t_stride = shared_t ? 0 : Nt;
    const bool gls = generalised != 0;
    size_t need;
    if (use_shared_path(h, t_stride, B, Nt, gls)) {
        const Plan pl = make_plan(h, B, Nt, Nf, 1);
        SharedLayout L;
        if (!shared_layout(pl, B, Nt, Nf, h->opt_table_mb << 20, L)) return LSP_EINVAL;
        need = L.total;
    } else {
        Route r;
        const int rc = route(h, t_stride, B, Nt, Nf, gls, r);
        if (rc != LSP_OK) return rc;
        need = device_layout(r.pl, B, Nt, Nf, r.tab_series, gls).total;
    }
    RefineList rl;                                        // (so that a call captured into a CUDA graph afterwards allocates nothing)
    if (h->opt_refine == 0) { const int rc = refine_list(h, rl); if (rc != LSP_OK) return rc; }
    return ensure(h, &h->buf, &h->buf_bytes, need);
}

int lsp_call_timing(lsp_handle h, int calls_back, float ms[4])
{
    if (!h || !ms || calls_back < 0) return LSP_EINVAL;
    if ((uint64_t)calls_back >= h->timed_calls || calls_back >= TIMING_RING) return LSP_EINVAL;
    DeviceGuard g(h->device);
    const int slot = (int)((h->timed_calls - 1 - (uint64_t)calls_back) % TIMING_RING);
    cudaEvent_t* ev = h->ev[slot];
    LSP_CUDA(h, cudaEventSynchronize(ev[4]));
    for (int i = 0; i < 4; ++i) LSP_CUDA(h, cudaEventElapsedTime(&ms[i], ev[i], ev[i + 1]));
    if (h->ev_chunks[slot] > 0) {                         // chunked call: accumulate = the accumulate launches only; the table pre-passes count as records
        float acc = 0.f, whole = 0.f;
        for (int c = 0; c < h->ev_chunks[slot]; ++c) {
            float d = 0.f;
            LSP_CUDA(h, cudaEventElapsedTime(&d, h->evc[slot][2 * c], h->evc[slot][2 * c + 1]));
            acc += d;
        }
        LSP_CUDA(h, cudaEventElapsedTime(&whole, ev[1], ev[3]));
        ms[1] = whole - acc; ms[2] = acc;
    }
    return LSP_OK;
}

int lsp_last_timing(lsp_handle h, float ms[4]) { return lsp_call_timing(h, 0, ms); }

int lsp_plan_query(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int64_t out[8])
{
    if (!out || sm_count < 1 || B < 1 || Nt < 2 || Nf < 1) return LSP_EINVAL;
    const PlanChoice pc = plan_choose(sm_count, B, Nt, Nf, PlanOverrides());
    out[0] = pc.K; out[1] = pc.T; out[2] = pc.nsplit; out[3] = pc.pipe;
    out[4] = pc.nfb; out[5] = pc.split_len; out[6] = pc.ctas_per_sm;
    out[7] = (int64_t)(pc.score * 1e6);
    return LSP_OK;
}

int lsp_plan_query_form(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int pipe, int64_t out[8])
{
    if (!out || sm_count < 1 || B < 1 || Nt < 2 || Nf < 1 || pipe < 0 || pipe > LSP_PIPE_TENSOR) return LSP_EINVAL;
    PlanOverrides ov;
    ov.pipe = pipe;
    const PlanChoice pc = plan_choose(sm_count, B, Nt, Nf, ov);
    out[0] = pc.K; out[1] = pc.T; out[2] = pc.nsplit; out[3] = pc.pipe;
    out[4] = pc.nfb; out[5] = pc.split_len; out[6] = (pc.pipe == PLAN_PIPE_TENSOR && pc.L >= 128) ? pc.nchunks : pc.ctas_per_sm;
    out[7] = (int64_t)plan_est_cycles(sm_count, B, Nt, Nf, pc);
    return LSP_OK;
}

int lsp_periodogram_batched(lsp_handle h,
                            const double* t, int64_t t_stride, const float* x, int64_t x_stride,
                            int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                            float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, void* stream)
{
    int rc = check_batch_args(h, t, x, B, Nt, 2, f_min, df, Nf, P, peak_idx, peak_val);
    if (rc == LSP_OK) rc = check_strides(t_stride, x_stride, p_stride, B, Nt, Nf, P);
    if (rc != LSP_OK) return rc;
    DeviceGuard g(h->device);
    return run_device(h, t, t_stride, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride,
                      peak_idx, peak_val, static_cast<cudaStream_t>(stream));
}

int lsp_periodogram_gls_batched(lsp_handle h,
                                const double* t, int64_t t_stride, const float* x, int64_t x_stride,
                                int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                                float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, void* stream)
{
    int rc = check_batch_args(h, t, x, B, Nt, 4, f_min, df, Nf, P, peak_idx, peak_val);
    if (rc == LSP_OK) rc = check_strides(t_stride, x_stride, p_stride, B, Nt, Nf, P);
    if (rc != LSP_OK) return rc;
    DeviceGuard g(h->device);
    return run_device(h, t, t_stride, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride,
                      peak_idx, peak_val, static_cast<cudaStream_t>(stream), true);
}

int lsp_periodogram_gls_weighted_batched(lsp_handle h,
                                         const double* t, int64_t t_stride, const float* x, int64_t x_stride,
                                         const float* w, int64_t w_stride,
                                         int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                                         float* P, int64_t p_stride, int32_t* peak_idx, float* peak_val, void* stream)
{
    int rc = check_batch_args(h, t, x, B, Nt, 4, f_min, df, Nf, P, peak_idx, peak_val);
    if (rc == LSP_OK) rc = check_strides(t_stride, x_stride, p_stride, B, Nt, Nf, P);
    if (rc == LSP_OK && w && B > 1 && w_stride != 0 && std::llabs(w_stride) < Nt) rc = LSP_EINVAL;
    if (rc != LSP_OK) return rc;
    DeviceGuard g(h->device);
    return run_device(h, t, t_stride, x, x_stride, B, Nt, f_min, df, Nf, P, p_stride,
                      peak_idx, peak_val, static_cast<cudaStream_t>(stream), true, w, w_stride);
}

int lsp_periodogram_gls_weighted(lsp_handle h, const double* t, const float* x, const float* w, int64_t Nt,
                                 double f_min, double df, int64_t Nf, float* P, void* stream)
{
    if (!P) return LSP_EINVAL;
    return lsp_periodogram_gls_weighted_batched(h, t, Nt, x, Nt, w, Nt, 1, Nt, f_min, df, Nf, P, Nf, nullptr, nullptr, stream);
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

// ---------------------------------------------------------------------------------------------------------------------------
// lsp_periodogram_static: one series through the FP32-pipe form with NO allocation of any kind -- for callers that cannot call
// cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  The workspace the other entry points
// keep in the handle's cudaMalloc'ed buffer (records, per-split partial sums, block partials, arg-max cell) lives instead in ONE
// file-scope device array of LSP_STATIC_SCRATCH_BYTES, which every GPU that loads this library holds until the process exits.
// In host code the array's NAME is only a host-side stand-in for the symbol, not a device address (a kernel given it would fault
// or, where the GPU can reach host memory, silently use the wrong memory): its address is resolved once per device, with that
// device current, by cudaGetSymbolAddress below, and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char lsp_static_scratch[LSP_STATIC_SCRATCH_BYTES];
static_assert(LSP_STATIC_MAX_NT <= REFINE_INPLACE_MAX_NT, "the static entry point relies on finish_kernel refining in place");
static_assert(2 * 16 * (int64_t)LSP_STATIC_MAX_NT + 4096 + 16 * (int64_t)LSP_STATIC_MAX_NF <= (int64_t)LSP_STATIC_SCRATCH_BYTES,
              "the stated limits must fit the array with one time split");

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
unsigned char* g_static_ptr[STATIC_MAX_DEVICES] = {};      // device address of lsp_static_scratch on device i (0: not resolved yet)
int g_static_sm[STATIC_MAX_DEVICES] = {};

// set-up, once per device (the calling thread's current device): no allocation, no synchronisation
int static_setup(int dev, unsigned char** ptr, int* sm_count)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        int major = 0, sms = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); return LSP_ECUDA; }
        if (major < 10 || sms < 1) return LSP_ECUDA;       // sm_100a SASS only: fail loudly elsewhere
        unsigned char* a = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&a, lsp_static_scratch);
        if (e != cudaSuccess || !a) { cudaGetLastError(); return LSP_ECUDA; }
        g_static_sm[dev] = sms;
        g_static_ptr[dev] = a;
    }
    *ptr = g_static_ptr[dev]; *sm_count = g_static_sm[dev];
    return LSP_OK;
}
}  // namespace

int lsp_periodogram_static(const double* t, const float* x, int64_t Nt, double f_min, double df, int64_t Nf,
                           float* P, int32_t* peak_idx, float* peak_val, void* stream)
{
    if (!t || !x || Nt < 2 || Nf < 1 || bad_grid(f_min, df)) return LSP_EINVAL;
    if ((peak_idx == nullptr) != (peak_val == nullptr) || (!P && !peak_idx)) return LSP_EINVAL;
    if (Nt > LSP_STATIC_MAX_NT || Nf > LSP_STATIC_MAX_NF) return LSP_ELIMIT;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return LSP_ECUDA; }
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return LSP_ELIMIT;
    unsigned char* base = nullptr; int sm_count = 0;
    int rc = static_setup(dev, &base, &sm_count);
    if (rc != LSP_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);

    // layout inside the array (every region is written in full by the call before it is read: nothing needs clearing but the
    // arg-max cell and its counter, which the records kernel resets)
    const int nparts = (int)((Nt + 511) / 512);                              // <= 32
    const int64_t part_chunk = (Nt + nparts - 1) / nparts;
    const size_t o_recA = 0;
    const size_t o_recB = align_up(o_recA + (size_t)Nt * sizeof(float4), 256);
    const size_t o_psum = align_up(o_recB + (size_t)Nt * sizeof(ulonglong2), 256);
    const size_t o_pvar = align_up(o_psum + (size_t)nparts * sizeof(double), 256);
    const size_t o_peak = align_up(o_pvar + (size_t)nparts * sizeof(double), 256);
    const size_t o_cnt = o_peak + 256;
    const size_t o_ws = o_cnt + 256;
    // the plan of the FP32-pipe form (no tunables apply), with as many time splits as the array has room for
    PlanOverrides ov;
    ov.pipe = PLAN_PIPE_FP32;
    PlanChoice pc = plan_choose_fp32(sm_count, 1, Nt, Nf, ov);
    const int64_t room = ((int64_t)LSP_STATIC_SCRATCH_BYTES - (int64_t)o_ws) / (16 * Nf);   // whole [4][Nf] float blocks
    if (room < 1) return LSP_ELIMIT;
    for (int64_t cap = room; pc.K && pc.nsplit > room && cap >= 1; --cap) { ov.nsplit = cap; pc = plan_choose_fp32(sm_count, 1, Nt, Nf, ov); }
    if (pc.K == 0 || pc.nsplit > room) return LSP_ELIMIT;
    const KernelEntry* ke = find_kernel(pc.K);
    if (!ke || pc.T < 32 || pc.T > ke->max_t || (pc.T % 32) != 0) return LSP_EINVAL;

    float4* recA = reinterpret_cast<float4*>(base + o_recA);
    ulonglong2* recB = reinterpret_cast<ulonglong2*>(base + o_recB);
    double* psum = reinterpret_cast<double*>(base + o_psum);
    double* pvar = reinterpret_cast<double*>(base + o_pvar);
    u64* peak64 = reinterpret_cast<u64*>(base + o_peak);
    unsigned* counter = reinterpret_cast<unsigned*>(base + o_cnt);
    float* ws = reinterpret_cast<float*>(base + o_ws);

    // steps 1-2 (the mean inside the records kernel: Nt <= 16,384; it also resets the arg-max cell and its counter)
    records_kernel<false, true><<<dim3((unsigned)nparts, 1u), 256, 0, st>>>(t, Nt, x, Nt, Nt, part_chunk, f_min, df, psum, recA, recB, pvar,
                                                                          peak64, counter, origin_offset(f_min, df, Nf), 1);
    if (cudaGetLastError() != cudaSuccess) return LSP_ECUDA;
    // steps 3-5
    const int flush_tiles = (int)((2048 + TILE_Z - 1) / TILE_Z);
    AccumParams ap;
    ap.recW = nullptr; ap.recA = recA; ap.recB = recB; ap.ws = ws; ap.ws1 = nullptr; ap.Nt = Nt; ap.Nf = Nf;
    ap.split_len = pc.split_len; ap.nsplit = pc.nsplit; ap.nfb = pc.nfb; ap.flush_tiles = flush_tiles;
    const bool direct = pc.split_len <= (int64_t)flush_tiles * TILE_Z;
    const size_t smem = accum_smem_bytes(ke, pc.T, false, direct);
    const accum_fn fn = direct ? ke->fn_direct : ke->fn;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return LSP_ECUDA; }
    fn<<<(unsigned)((int64_t)pc.nsplit * pc.nfb), pc.T, smem, st>>>(ap);
    if (cudaGetLastError() != cudaSuccess) return LSP_ECUDA;
    // steps 6-7; ill-conditioned frequencies are redone in fp64 inside finish_kernel (Nt <= 16,384: no list, no further kernel)
    FinishParams fp;
    fp.ws = ws; fp.part_var = pvar; fp.P = P; fp.p_stride = Nf;
    fp.peak_idx = peak_idx; fp.peak_val = peak_val; fp.peak64 = peak64; fp.counter = counter;
    fp.Nt = Nt; fp.Nf = Nf; fp.nsplit = pc.nsplit; fp.nparts = nparts;
    fp.x_scaled = 0; fp.ws1 = nullptr; fp.ws_x = nullptr; fp.x_row = 0;
    fp.src.t = t; fp.src.t_stride = Nt; fp.src.x = x; fp.src.x_stride = Nt; fp.src.w = nullptr; fp.src.w_stride = 0;
    fp.src.f_min = f_min; fp.src.df = df; fp.src.Nt = Nt;
    fp.refine_amp = refine_amplification(false, Nt, false); fp.refine_pow = INFINITY;
    fp.list = RefineList{};
    launch_finish(fp, 1, st);
    if (cudaGetLastError() != cudaSuccess) return LSP_ECUDA;
    return LSP_OK;
}

int lsp_periodogram_batched_host(lsp_handle h, const double* t, int share_t, const float* x,
                                 int64_t B, int64_t Nt, double f_min, double df, int64_t Nf,
                                 float* P, int32_t* peak_idx, float* peak_val, void* stream)
{
    const int rc0 = check_batch_args(h, t, x, B, Nt, 2, f_min, df, Nf, P, peak_idx, peak_val);
    if (rc0 != LSP_OK) return rc0;
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
    // Large batches: the series are independent, so the call is pipelined over chunks of series -- the H2D copy of chunk c+1 and
    // the D2H copy of chunk c-1 run on two copy streams while chunk c computes on `stream` (same kernels, same results).
    const int nchunk = host_pipe_chunks(h, share_t != 0, B, Nt, Nf, P != nullptr);
    h->last_host_chunks = nchunk;
    if (nchunk > 1) {
        if (!h->s_in) LSP_CUDA(h, cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
        if (!h->s_out) LSP_CUDA(h, cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
        for (cudaEvent_t& e : h->ev_pipe) if (!e) LSP_CUDA(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        cudaEvent_t e_start = h->ev_pipe[2 * HOST_PIPE_CHUNKS];
        LSP_CUDA(h, cudaEventRecord(e_start, st));                    // earlier work on `stream` may still use the staging buffers
        LSP_CUDA(h, cudaStreamWaitEvent(h->s_in, e_start, 0));
        LSP_CUDA(h, cudaStreamWaitEvent(h->s_out, e_start, 0));
        const int64_t per = (B + nchunk - 1) / nchunk;
        if (share_t) LSP_CUDA(h, cudaMemcpyAsync(d_t, t, nt_t * sizeof(double), cudaMemcpyHostToDevice, h->s_in));
        for (int c = 0; c < nchunk; ++c) {                            // all copies in, back to back
            const int64_t b0 = c * per, nb = (B - b0 < per) ? B - b0 : per;
            if (nb <= 0) break;
            if (!share_t) LSP_CUDA(h, cudaMemcpyAsync(d_t + b0 * Nt, t + b0 * Nt, (size_t)nb * Nt * sizeof(double), cudaMemcpyHostToDevice, h->s_in));
            LSP_CUDA(h, cudaMemcpyAsync(d_x + b0 * Nt, x + b0 * Nt, (size_t)nb * Nt * sizeof(float), cudaMemcpyHostToDevice, h->s_in));
            LSP_CUDA(h, cudaEventRecord(h->ev_pipe[c], h->s_in));
        }
        for (int c = 0; c < nchunk; ++c) {
            const int64_t b0 = c * per, nb = (B - b0 < per) ? B - b0 : per;
            if (nb <= 0) break;
            LSP_CUDA(h, cudaStreamWaitEvent(st, h->ev_pipe[c], 0));
            rc = run_device(h, share_t ? d_t : d_t + b0 * Nt, share_t ? 0 : Nt, d_x + b0 * Nt, Nt, nb, Nt, f_min, df, Nf,
                            d_P ? d_P + b0 * Nf : nullptr, Nf, d_pi ? d_pi + b0 : nullptr, d_pv ? d_pv + b0 : nullptr, st);
            if (rc != LSP_OK) { cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(h->s_out); cudaStreamSynchronize(st); return rc; }
            LSP_CUDA(h, cudaEventRecord(h->ev_pipe[HOST_PIPE_CHUNKS + c], st));
            LSP_CUDA(h, cudaStreamWaitEvent(h->s_out, h->ev_pipe[HOST_PIPE_CHUNKS + c], 0));
            if (P) LSP_CUDA(h, cudaMemcpyAsync(P + b0 * Nf, d_P + b0 * Nf, (size_t)nb * (size_t)Nf * sizeof(float), cudaMemcpyDeviceToHost, h->s_out));
            if (peak_idx) {
                LSP_CUDA(h, cudaMemcpyAsync(peak_idx + b0, d_pi + b0, (size_t)nb * sizeof(int32_t), cudaMemcpyDeviceToHost, h->s_out));
                LSP_CUDA(h, cudaMemcpyAsync(peak_val + b0, d_pv + b0, (size_t)nb * sizeof(float), cudaMemcpyDeviceToHost, h->s_out));
            }
        }
        LSP_CUDA(h, cudaStreamSynchronize(h->s_out));
        LSP_CUDA(h, cudaStreamSynchronize(st));
        return LSP_OK;
    }
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

int lsp_probe_mma_accumulate(lsp_handle h, float out[8])
{
    if (!h || !out) return LSP_EINVAL;
    DeviceGuard g(h->device);
    // start value 2^24 + 2 (ulp 2), built exactly by two MMAs; then one more MMA with the products listed
    const float big[2] = {4096.f, 4096.f}, two[2] = {2.f, 1.f};
    const float third[8][PROBE_MAX_PRODUCTS] = {
        {0.f, 0.f, 0.f, 0.f},                       // [0] nothing:                 2^24 + 2
        {1.f, 0.f, 0.f, 0.f},                       // [1] + 1  (half an ulp):      truncation keeps 2^24 + 2 (rounding would give 2^24 + 4)
        {-1.f, 0.f, 0.f, 0.f},                      // [2] - 1:                     2^24
        {-0.5f, 0.f, 0.f, 0.f},                     // [3] - 0.5 (a quarter ulp):   2^24: within the two extra bits, pulls a whole ulp
        {-0.0009765625f, 0.f, 0.f, 0.f},            // [4] - 2^-10:                 2^24 + 2: below the extra bits, dropped
        {-0.75f, -0.75f, -0.75f, -0.75f},           // [5] four times - 0.75:       2^24 (each product cut to - 0.5 first; the exact sum is 2^24 - 1)
        {0.75f, 0.75f, 0.75f, 0.75f},               // [6] four times + 0.75:       2^24 + 4
        {3.f, 0.f, 0.f, 0.f},                       // [7] + 3:                     2^24 + 4 (exact 2^24 + 5 truncated)
    };
    ProbeSeq host[8];
    for (int s = 0; s < 8; ++s) {
        ProbeSeq q = {};
        q.n = 3;
        q.a[0][0] = big[0]; q.b[0][0] = big[1]; q.a[1][0] = two[0]; q.b[1][0] = two[1];
        for (int k = 0; k < PROBE_MAX_PRODUCTS; ++k) { q.a[2][k] = third[s][k]; q.b[2][k] = 1.f; }
        host[s] = q;
    }
    ProbeSeq* d_seq = nullptr; float* d_out = nullptr;
    LSP_CUDA(h, cudaMalloc(&d_seq, sizeof(host)));
    cudaError_t e = cudaMalloc(&d_out, 8 * sizeof(float));
    if (e != cudaSuccess) { cudaFree(d_seq); return cuda_fail(h, e); }
    e = cudaMemcpy(d_seq, host, sizeof(host), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) { probe_mma_kernel<<<1, 128, 8192>>>(d_seq, 8, d_out); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaMemcpy(out, d_out, 8 * sizeof(float), cudaMemcpyDeviceToHost);
    cudaFree(d_seq); cudaFree(d_out);
    return e == cudaSuccess ? LSP_OK : cuda_fail(h, e);
}

int lsp_last_plan(lsp_handle h, int64_t out[8])
{
    if (!h || !out) return LSP_EINVAL;
    const Plan& p = h->plan;
    out[0] = p.K; out[1] = p.T; out[2] = p.nsplit; out[3] = p.pipe;
    out[4] = p.nfb; out[5] = p.split_len; out[6] = p.launches;
    out[7] = (p.pipe == PLAN_PIPE_TENSOR) ? 0 : 6;        // 0: tensor-core form (16 tensor FLOP per term)
    return LSP_OK;
}

const char* lsp_last_kernel_name(lsp_handle h) { return h ? h->plan.kernel_name : ""; }

int lsp_last_host_chunks(lsp_handle h) { return h ? h->last_host_chunks : 0; }

int lsp_last_cuda_error(lsp_handle h) { return h ? h->last_cuda : 0; }

const char* lsp_status_string(int status)
{
    switch (status) {
        case LSP_OK:     return "ok";
        case LSP_EINVAL: return "invalid argument";
        case LSP_ECUDA:  return "CUDA runtime error (or no sm_100 device)";
        case LSP_ENOMEM: return "device workspace allocation failed";
        case LSP_ELIMIT: return "size beyond the fixed limits of lsp_periodogram_static (Nt <= 16,384, Nf <= 262,144)";
        default:         return "unknown status";
    }
}

const char* lsp_version(void) { return "lsp_b200 0.2 (sm_100a)"; }

}  // extern "C"
