/*
 * lsp.h -- C ABI of the B200-native direct Lomb-Scargle periodogram library.
 *
 * The operation (Townsend 2010, arxiv 1007.1658; line numbers are /root/reference/PAPER.md):
 * for a time series (t_j, x_j), j = 0..Nt-1, shifted and scaled to zero mean and unit
 * variance, and a uniform frequency grid f_k = f_min + k*df, k = 0..Nf-1
 * (eq. (9), generalised to a free f_min), compute the normalised periodogram
 *
 *     P(f) = 1/2 { [sum_j X_j cos w(t_j - tau)]^2 / sum_j cos^2 w(t_j - tau)
 *                + [sum_j X_j sin w(t_j - tau)]^2 / sum_j sin^2 w(t_j - tau) },   w = 2 pi f   (eq. 1)
 *     tan 2 w tau = sum_j sin 2 w t_j / sum_j cos 2 w t_j                                        (eq. 2)
 *
 * evaluated through the single-pass sums XC, XS, CC, CS of eqs (5)-(8) with
 * SS = Nt - CC.  X_j = x_j - mean(x); the variance is the sample variance
 * sum X_j^2 / (Nt - 1) (reading G1).  Cost is O(Nt*Nf) "term evaluations" (eq. 4).
 *
 * Conventions
 *   - Pointers marked DEVICE are CUDA device pointers on the handle's device; pointers marked
 *     HOST are ordinary (pageable or pinned) host pointers.  The caller owns every array; the
 *     library never frees or reallocates caller memory.  The handle owns a device workspace
 *     that grows to the largest call seen (growth allocates and may synchronise the device once;
 *     lsp_reserve sizes it ahead of time).  Size: 32 B per sample + 16 B x Nf x (time splits, <= 2 GiB)
 *     + at most LSP_PARAM_TABLE_MB for the tensor form's table (+ 8.5 MiB, once, for the list of LSP_PARAM_REFINE);
 *     if it cannot be allocated the call returns LSP_ENOMEM and the handle keeps the workspace it had.
 *   - Device-pointer entry points only ENQUEUE work on `stream` (a cudaStream_t passed as
 *     void*; NULL = legacy default stream) and return without synchronising; inputs must stay
 *     valid until the stream reaches the end of the call.  Host-pointer entry points copy
 *     in, compute, copy out and synchronise `stream` before returning.
 *   - One handle serves one stream at a time (the workspace is not shared between concurrent calls).
 *   - t and 1/f share a unit (days and cycles/day in the paper's workloads).  Times need not be sorted.
 *   - Return value: LSP_OK (0) or a negative LSP_E* code; nothing throws, nothing aborts.
 *     Data-dependent degeneracy (zero variance) cannot be reported without a sync: P is NaN then.
 *   - f = 0 is legal: the sine term of eq. (1) is 0/0 and dropped (reading G7), P = XC^2/Nt/(2 var) ~ 0.
 *   - Accuracy: max |P - P_fp64| <= 1e-4 max P on any grid, including f T << 1 and the aliases of regular sampling, where the
 *     single-pass sums of eqs (5)-(8) are ill-conditioned (R -> Nt): those frequencies are recomputed from t and x in fp64
 *     (LSP_PARAM_REFINE; DESIGN.md section 6 item 6); verified from Nt = 2 up.  The tensor form forced below Nt = 512
 *     (LSP_PARAM_PIPE = 2; the automatic plan never picks it there) is good to 5e-3 only.
 *   - There is no CPU fallback: without a CUDA device lsp_create fails with LSP_ECUDA.
 */
#ifndef LSP_B200_H
#define LSP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lsp_ctx* lsp_handle;            /* opaque; owns the device workspace only */

enum {
    LSP_OK      =  0,
    LSP_EINVAL  = -1,   /* NULL handle/pointer, Nt < 2, Nf < 1, B < 1 or B > 65,535, bad stride, non-finite or negative f_min/df */
    LSP_ECUDA   = -2,   /* a CUDA runtime call failed; see lsp_last_cuda_error */
    LSP_ENOMEM  = -3,   /* workspace allocation failed */
    LSP_ELIMIT  = -4    /* lsp_periodogram_static only: Nt or Nf beyond its fixed limits */
};

/*
 * Tunables for lsp_set_param (all optional; 0 restores the automatic choice).  Steps 3-5 of the path (anchor, rotate and
 * accumulate, cascade: the O(Nt*Nf) part) exist in two forms that compute the same sums of eq. (8):
 *   LSP_PIPE_FP32    the paper's arithmetic: fp32 throughout, SFU sin/cos at anchors,
 *                    K adjacent frequencies per thread advanced by a re-anchored three-term recurrence; 6 FP32 lane-ops per term.
 *   LSP_PIPE_TENSOR  the same recurrence (angle addition) factorised over a uniform grid into a dense contraction and run
 *                    on the tensor cores with fp16 hi + lo operands (22 bits; by default the two small cross products share
 *                    one e5m2 MMA) and fp32 accumulation; about ten times faster, within the 1e-4 max P tolerance of the path.
 * Automatic: the tensor form when Nt >= 512 and the cost model says it is faster.
 */
enum {
    LSP_PARAM_K         = 1,  /* FP32 form: adjacent frequencies per thread: 4, 8, ..., 32 */
    LSP_PARAM_THREADS   = 2,  /* FP32 form: threads per CTA: 32..256 (multiple of 32; <= 128 for K >= 28) */
    LSP_PARAM_NSPLIT    = 3,  /* number of time-axis splits per (series, frequency block) */
    LSP_PARAM_PIPE      = 4,  /* LSP_PIPE_FP32 or LSP_PIPE_TENSOR (see above) */
    LSP_PARAM_FLUSH     = 5,  /* samples between folds of the fp32 partial sums / drains of the TMEM accumulators (default 2,048; CTA-pair form 4,096) */
    LSP_PARAM_TIMING    = 6,  /* 1 = record CUDA events around each kernel of a call (see lsp_last_timing) */
    LSP_PARAM_TABLE_MB  = 7,  /* tensor form, CTA-pair kernel: MiB of workspace its operand table may take (default 1,024);  */
                              /* a series whose table (3 KB per sample) is larger runs in time chunks, same result             */
    LSP_PARAM_COARSE    = 8,  /* tensor form: coarse extent L = 16, 32, 64 (a CTA owns 128 L frequencies) or 128 (CTA pairs,   */
                              /* 32,768 frequencies per pair, one operand streamed from the table)                             */
    LSP_PARAM_TRUNC     = 9,  /* tensor forms: 1 = do not add the expected round-toward-zero loss of the tensor-core          */
                              /* accumulation back at each drain; 0 = add it (default); CTA-pair kernel   */
                              /* also n > 1: a fixed n / 1000 ulps per 8 samples instead of the model (ablation)                */
    LSP_PARAM_SHARED    = 11, /* batched call with t_stride = 0: 0 = the shared-time GEMM path when B >= 16 and Nt >= 512, 1 = never, 2 = always */
    LSP_PARAM_CORR      = 15, /* tensor form, CTA-pair kernel: how the first-order corrections A_lo B_hi + A_hi B_lo of the fp16 hi + lo   */
                              /* operand split are formed: 0 = one kind::f8f6f4 MMA on e5m2 copies (3 MMAs per 8 samples, the default);  */
                              /* 1 = two kind::f16 MMAs on fp16 lo parts (4 MMAs per 8 samples): every product of the sums XC, XS then   */
                              /* carries 22 significant operand bits, no less than the paper's fp32 arithmetic with SFU trig*/
    LSP_PARAM_REFINE    = 16, /* 0 = frequencies whose sums are ill-conditioned (R > 0.8 Nt in eq. (5) on the FP32-pipe form, R > 0.45 Nt  */
                              /* on the tensor-core forms, less below 1,000 samples: f T << 1 and the aliases of regular sampling; the     */
                              /* generalised form by its determinant) are recomputed from the raw series in fp64, and on the tensor-core  */
                              /* forms also the frequencies of strong lines (P > 0.0118 Nt, i.e. 2.4 % of the largest possible power)      */
                              /* (default; none on a grid that starts at 1/T over irregular times of noise); 1 = keep the value of the      */
                              /* fp32 sums there (poor below f T ~ 0.5 on the tensor forms)                                               */
    LSP_PARAM_ORDER     = 17, /* tensor-core forms: 0 = the per-sample records are laid out in a golden-ratio stride order, so that every      */
                              /* accumulation window holds samples from all over the time span (a strong trend or slow signal, inside the   */
                              /* grid or below it, then no longer makes the tensor core's truncating accumulator swing: DESIGN.md section   */
                              /* 8) (default); 1 = in the order given                                                                      */
    LSP_PARAM_PDL       = 13  /* short-grid tensor path: 0 = steps 1-2 run inside the accumulate kernel when Nt <= 16,384 (two launches per  */
                              /* call) and the kernels of a call are launched as programmatic dependents (each kernel's launch and      */
                              /* set-up overlap its predecessor's tail); 1 = separate pre-pass kernels in plain stream order            */
};
enum { LSP_PIPE_AUTO = 0, LSP_PIPE_FP32 = 1, LSP_PIPE_TENSOR = 2 };
/* lsp_periodogram_static: its fixed device array and the sizes it accepts */
enum { LSP_STATIC_SCRATCH_BYTES = 8 << 20, LSP_STATIC_MAX_NT = 16384, LSP_STATIC_MAX_NF = 262144 };

/* Create a handle bound to CUDA device `device` (-1 = the calling thread's current device). */
int lsp_create(lsp_handle* out, int device);

/* Free the workspace and the handle.  NULL is accepted.  Synchronises the device. */
int lsp_destroy(lsp_handle h);

/* Override / query a tunable (see LSP_PARAM_*).  Returns LSP_EINVAL for unknown keys or values. */
int lsp_set_param(lsp_handle h, int key, int64_t value);
int lsp_get_param(lsp_handle h, int key, int64_t* value);

/*
 * One series.  P[k] = P(f_min + k*df), k = 0..Nf-1  (eqs (1)-(2) via (5)-(8)).
 *   t  DEVICE const double[Nt]   sample times
 *   x  DEVICE const float [Nt]   measurements (any mean / variance; normalised inside)
 *   P  DEVICE       float [Nf]   written; exactly Nf values (reading G8: no rounding up to blocks)
 * Enqueues 3-5 kernels on `stream` (more when the series runs in time chunks; lsp_last_plan reports how many); no host
 * synchronisation, no allocation once the workspace has grown to the problem size (lsp_reserve): the call can be captured
 * into a CUDA graph.
 */
int lsp_periodogram(lsp_handle h,
                    const double* t, const float* x, int64_t Nt,
                    double f_min, double df, int64_t Nf,
                    float* P, void* stream);

/*
 * B independent series on one shared frequency grid (the Monte-Carlo use of PAPER.md:369).
 *   series b reads t + b*t_stride and x + b*x_stride (strides in ELEMENTS; t_stride = 0 means
 *   all series share one time vector; otherwise |stride| >= Nt), writes P + b*p_stride.  1 <= B <= 65,535.
 *   With t_stride = 0 (the Monte-Carlo use: sampling kept, noise redrawn) and B >= 16, Nt >= 512 the sums sum_j X_bj cos / sin
 *   are evaluated as ONE dense contraction over all series and CC, CS once per frequency (same result, ~5x faster).
 *   P may be NULL if only the peaks are wanted (then p_stride is ignored).
 *   peak_idx DEVICE int32[B], peak_val DEVICE float[B]: arg-max_k P (lowest k among equal
 *   maxima, reading G9) and its value; both nullable (both or neither).
 */
int lsp_periodogram_batched(lsp_handle h,
                            const double* t, int64_t t_stride,
                            const float* x, int64_t x_stride,
                            int64_t B, int64_t Nt,
                            double f_min, double df, int64_t Nf,
                            float* P, int64_t p_stride,
                            int32_t* peak_idx, float* peak_val,
                            void* stream);

/*
 * Generalised (floating-mean) periodogram -- the extension the paper names in section 6.3 (Zechmeister &
 * Kuerster 2009): for every frequency the least-squares fit x_j ~ a cos(w t_j) + b sin(w t_j) + c, returned as
 * P = (chi0^2 - chi^2_min) / (2 var) -- the normalisation of eq. (1), to which it reduces when the constant is
 * orthogonal to the sinusoids.  Same arguments, layout, ownership and errors as lsp_periodogram[_batched], Nt >= 4.
 * Computed from the sums of eq. (8) plus sum cos(w t_j), sum sin(w t_j), which a second accumulate pass with unit
 * weights provides (cost: two accumulate launches on the tensor-core forms, one on the FP32-pipe form).  Where the fit is singular (f -> 0: D = CCn SSn - CSn^2 <= 1e-9) P = 0.
 */
int lsp_periodogram_gls(lsp_handle h,
                        const double* t, const float* x, int64_t Nt,
                        double f_min, double df, int64_t Nf,
                        float* P, void* stream);

int lsp_periodogram_gls_batched(lsp_handle h,
                                const double* t, int64_t t_stride,
                                const float* x, int64_t x_stride,
                                int64_t B, int64_t Nt,
                                double f_min, double df, int64_t Nf,
                                float* P, int64_t p_stride,
                                int32_t* peak_idx, float* peak_val,
                                void* stream);

/*
 * Weighted generalised periodogram (the per-sample weights of Zechmeister & Kuerster 2009):
 * the fit of lsp_periodogram_gls with chi^2 = sum_j w_j (x_j - a cos - b sin - c)^2, returned as
 *     P = (Nt - 1)/2 * (chi0^2 - chi^2_min) / chi0^2,   chi0^2 = sum_j w_j (x_j - xbar_w)^2,  xbar_w = sum w x / sum w
 * (reading G14: the unweighted normalisation written as a chi^2 ratio; w_j = const gives
 * lsp_periodogram_gls; 0 <= P <= (Nt - 1)/2).  Typical use: w_j = 1 / sigma_j^2.
 *   w DEVICE const float[Nt] per series (series b at w + b*w_stride, |w_stride| >= Nt; w_stride = 0: one weight vector for
 *   all series), finite, >= 0, positive sum (not checked: a violation yields NaN).  Only weight ratios matter; w_j = 0
 *   removes sample j from the fit.  w == NULL: unit weights (identical to lsp_periodogram_gls[_batched]).
 *   Everything else as lsp_periodogram_gls[_batched].  Two accumulate passes in whatever form the plan picks: on the tensor-core
 *   forms the generated operand carries w_j x_j, and w_j e^{2i theta} for the sums of cos^2, cos sin; on the FP32 pipe the samples
 *   enter as sqrt(w_j) x_j and sqrt(w_j) e^{i theta} (the recurrence is linear, so the weights cost nothing per term).
 */
int lsp_periodogram_gls_weighted(lsp_handle h,
                                 const double* t, const float* x, const float* w, int64_t Nt,
                                 double f_min, double df, int64_t Nf,
                                 float* P, void* stream);

int lsp_periodogram_gls_weighted_batched(lsp_handle h,
                                         const double* t, int64_t t_stride,
                                         const float* x, int64_t x_stride,
                                         const float* w, int64_t w_stride,
                                         int64_t B, int64_t Nt,
                                         double f_min, double df, int64_t Nf,
                                         float* P, int64_t p_stride,
                                         int32_t* peak_idx, float* peak_val,
                                         void* stream);

/*
 * Host-buffer forms: same arithmetic, HOST pointers.  The call copies t and x to the device
 * (cudaMemcpyAsync), runs the device path, copies P (and the peaks) back and synchronises
 * `stream`.  Arrays are dense: series b at t + b*Nt, x + b*Nt, P + b*Nf.
 * share_t != 0: t holds ONE time vector of length Nt used by every series.
 * Batches of >= 64 series that move >= 8 MiB are pipelined over 2 or 4 chunks of series: the copies of a chunk run on two
 * copy streams owned by the handle while its neighbours compute on `stream` (same kernels, same results; pinned host
 * buffers are needed for the copies to overlap).
 */
int lsp_periodogram_host(lsp_handle h,
                         const double* t, const float* x, int64_t Nt,
                         double f_min, double df, int64_t Nf,
                         float* P, void* stream);

int lsp_periodogram_batched_host(lsp_handle h,
                                 const double* t, int share_t, const float* x,
                                 int64_t B, int64_t Nt,
                                 double f_min, double df, int64_t Nf,
                                 float* P, int32_t* peak_idx, float* peak_val,
                                 void* stream);

/*
 * False-alarm probability, eq. (3):  Q[i] = 1 - [1 - (1 - p_i)^((Nt-3)/2)]^N_ind,  p_i = 2 P[i]/(Nt - 1)
 * for n periodogram values (a whole periodogram, or the per-series peaks of a batch).  p is the paper's 2 P_n/N_t: the beta
 * variable of PAPER.md:50 written for the sample-variance scaling this library uses (readings G1, G13).
 *   P DEVICE const float[n] (normalised power, as written by lsp_periodogram*), Q DEVICE float[n] (may alias P).
 *   Nt >= 4: samples of the series that produced P;  N_ind >= 1: number of independent frequencies -- the paper's
 *   N_f, or the N_f,ind <= N_f of PAPER.md:369 (real-valued).  Enqueues one kernel on `stream`; no synchronisation.
 */
int lsp_false_alarm(lsp_handle h, const float* P, int64_t n, int64_t Nt, double N_ind, float* Q, void* stream);

/*
 * One series, NO ALLOCATION: for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it).  Same result as lsp_periodogram with LSP_PARAM_PIPE = LSP_PIPE_FP32 (eqs (1)-(2) via (5)-(8),
 * the paper's fp32 arithmetic, ill-conditioned frequencies refined in fp64), plus the optional peak of
 * lsp_periodogram_batched.  No handle: it runs on the calling thread's CURRENT device; no tunables apply.
 *   t DEVICE const double[Nt], x DEVICE const float[Nt], P DEVICE float[Nf] (nullable if the peak is asked for),
 *   peak_idx DEVICE int32_t[1], peak_val DEVICE float[1] (both or neither; lowest index among equal maxima, reading G9).
 * Limits: 2 <= Nt <= LSP_STATIC_MAX_NT (16,384), 1 <= Nf <= LSP_STATIC_MAX_NF (262,144); beyond them LSP_ELIMIT, nothing launched.
 * Its workspace (32 B per sample + 16 B x Nf x time splits, as many splits as fit) is a file-scope `static __device__` array of
 * LSP_STATIC_SCRATCH_BYTES (8 MiB) inside the library: every GPU that loads the library holds those 8 MiB until the process
 * exits.  The call itself calls no cudaMalloc / cudaFree and no allocating library routine, never synchronises, and enqueues
 * three kernels on `stream`; the first call on a device also resolves the array's device address (cudaGetSymbolAddress).
 * ALL calls on a device share the one array, which keeps the previous call's contents: every region is rewritten before it is
 * read and the arg-max cell is reset by the call's first kernel, so calls in stream order are independent of each other --
 * but two calls that OVERLAP on the GPU (different streams, or graphs replayed concurrently) race on it: serialise them.
 */
int lsp_periodogram_static(const double* t, const float* x, int64_t Nt, double f_min, double df, int64_t Nf,
                           float* P, int32_t* peak_idx, float* peak_val, void* stream);

/*
 * Grow the workspace now to what a call with (B series -- `shared_t` != 0: on one time vector --, Nt samples, Nf
 * frequencies, generalised or not) needs under the handle's current tunables, so that the call itself allocates nothing
 * (CUDA-graph capture, latency-critical first calls).  May synchronise the device.  LSP_ENOMEM leaves the workspace as it was.
 */
int lsp_reserve(lsp_handle h, int64_t B, int shared_t, int64_t Nt, int64_t Nf, int generalised);

/*
 * Introspection of the last call's launch plan (for benchmarks and tests): fills
 * out[0..7] = {K (FP32 form) or L (tensor form), threads, nsplit, pipe (LSP_PIPE_*), n_freq_blocks, split_len, launches,
 *              FP32 lane-ops per term (6; 0 for the tensor form: 16 tensor FLOP per term)}.
 */
int lsp_last_plan(lsp_handle h, int64_t out[8]);

/*
 * Per-kernel device time of the last call, from CUDA events recorded on the call's stream
 * (only when LSP_PARAM_TIMING is 1).  Synchronises on the last event.
 * ms[0..3] = {moments, records, accumulate, finish} in milliseconds.
 */
int lsp_last_timing(lsp_handle h, float ms[4]);

/*
 * Same for an earlier call: calls_back = 0 is the last timed call, 1 the one before, ... up to
 * 63 (the handle keeps a ring of 64 event sets), so a benchmark can time many back-to-back
 * calls without a host synchronisation between them.  LSP_EINVAL if that call is not in the ring.
 */
int lsp_call_timing(lsp_handle h, int calls_back, float ms[4]);

/*
 * Host-only: the launch plan the library would pick for (B series, Nt samples, Nf frequencies) on a
 * device with `sm_count` SMs.  Needs no GPU.  out[0..7] = {K or L, threads, nsplit, pipe,
 * n_freq_blocks, split_len, resident CTAs per SM, model score * 1e6}.
 */
int lsp_plan_query(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int64_t out[8]);

/*
 * Same for one form of steps 3-5: pipe = LSP_PIPE_AUTO (identical to lsp_plan_query), LSP_PIPE_FP32 or LSP_PIPE_TENSOR.
 * For the tensor form K is reported as the coarse extent L (16, 32, 64, 128), a frequency block is 128 L frequencies and
 * `threads` is the CTA size (288 for L < 128, 544 for L = 128).  out[6] = time chunks (tensor form, L = 128) or resident CTAs
 * per SM (otherwise); out[7] = estimated SM cycles of the accumulate kernels (the quantity the automatic choice compares).
 */
int lsp_plan_query_form(int sm_count, int64_t B, int64_t Nt, int64_t Nf, int pipe, int64_t out[8]);

/* Name of the accumulate kernel the last call launched (static string; "" before any call). */
const char* lsp_last_kernel_name(lsp_handle h);

/*
 * Hardware check behind the tensor forms' truncation compensation: runs eight one-element tcgen05.mma
 * sequences on the device (synchronous, default stream) and returns the accumulator after each.  Start value 2^24 + 2 (ulp 2), then
 * one more MMA adding: out[0] nothing, [1] +1, [2] -1, [3] -0.5, [4] -2^-10, [5] four products of -0.75, [6] four of +0.75, [7] +3.
 * Measured on B200: {16777218, 16777218, 16777216, 16777216, 16777218, 16777216, 16777220, 16777220} -- products and accumulator
 * aligned with two extra bits, each truncated toward zero, the sum truncated toward zero.  HOST out[8].
 */
int lsp_probe_mma_accumulate(lsp_handle h, float out[8]);

/* Chunks of series the last host-buffer batched call was pipelined over (1: not pipelined; 0 before any such call). */
int lsp_last_host_chunks(lsp_handle h);

/* Last cudaError_t seen by the handle (0 = cudaSuccess). */
int lsp_last_cuda_error(lsp_handle h);

/* Human-readable text for a status code. */
const char* lsp_status_string(int status);

/* Library version string, e.g. "lsp_b200 0.2 (sm_100a)". */
const char* lsp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LSP_B200_H */
