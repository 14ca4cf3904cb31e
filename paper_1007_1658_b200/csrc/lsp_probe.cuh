// lsp_probe.cuh -- a check of the one hardware behaviour the tensor forms' truncation compensation rests on (tc_trunc_comp,
// lsp_tc.cuh): how tcgen05.mma kind::f16 folds products into its fp32 accumulator.  One CTA issues short
// sequences of MMAs whose only non-zero products sit on output element (0, 0) and returns that element after each sequence.
// On B200 (measured, round 2): the products of an output element and the accumulator are aligned to the largest exponent among
// them with two extra bits, each truncated toward zero, summed, and the sum truncated toward zero to fp32.
#pragma once
#include "lsp_tc.cuh"

namespace lsp {

constexpr int PROBE_MAX_MMAS = 4, PROBE_MAX_PRODUCTS = 4;
struct ProbeSeq { int n; float a[PROBE_MAX_MMAS][PROBE_MAX_PRODUCTS]; float b[PROBE_MAX_MMAS][PROBE_MAX_PRODUCTS]; };
constexpr uint32_t PROBE_IDESC = umma_idesc(128, 16);

// <<<1, 128, 8192>>>: out[s] = D[0][0] after the MMAs of seqs[s] (MMA i accumulates onto MMA i - 1; the first one overwrites)
__global__ void __launch_bounds__(128) probe_mma_kernel(const ProbeSeq* seqs, int nseq, float* out)
{
    extern __shared__ __align__(128) unsigned char probe_smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_slot;
    const unsigned tid = threadIdx.x, w = tid >> 5;
    const uint32_t sA = smem_u32(probe_smem), sB = sA + 4096;           // A: 128 rows x 16 fp16, B: 16 rows x 16 fp16, no-swizzle K-major
    if (tid == 0) { mbar_init(smem_u32(&bar), 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    if (w == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_slot)), "r"(32u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before(); __syncthreads(); tc_fence_after();
    const uint32_t tmem = tmem_slot;
    uint32_t phase = 0;
    for (int s = 0; s < nseq; ++s) {
        const ProbeSeq q = seqs[s];
        for (int i = 0; i < q.n; ++i) {
            for (int x = tid; x < (4096 + 512) / 4; x += 128) reinterpret_cast<uint32_t*>(probe_smem)[x] = 0u;
            __syncthreads();
            if (tid == 0) {                                             // row 0, K = 0..3 of both operands: the first 8 bytes of each tile
                __half* A = reinterpret_cast<__half*>(probe_smem);
                __half* B = reinterpret_cast<__half*>(probe_smem + 4096);
                for (int k = 0; k < PROBE_MAX_PRODUCTS; ++k) { A[k] = __float2half(q.a[i][k]); B[k] = __float2half(q.b[i][k]); }
            }
            fence_proxy_async();
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
                tc_mma_f16(tmem, umma_desc(sA, 2048, 128), umma_desc(sB, 256, 128), PROBE_IDESC, i > 0 ? 1u : 0u);
                tc_commit(smem_u32(&bar));
            }
            mbar_wait(smem_u32(&bar), phase); phase ^= 1u;
            tc_fence_after();
            __syncthreads();
        }
        float v[8];
        tmem_ld8(tmem + ((32u * w) << 16), v);
        if (tid == 0) out[s] = v[0];
        tc_fence_before();
        __syncthreads();
    }
    if (w == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(32u) : "memory");
}

}  // namespace lsp
