// lsp_common.cuh -- shared device helpers and data layout of the B200 Lomb-Scargle path.
//
// Layout in HBM (all owned by the handle's workspace):
//   recA[B][Nt]  float4     {X_j, cos d_j, sin d_j, 2 cos d_j}   X_j = x_j - mean; d_j = 2 pi frac(df * t'_j)
//   recB[B][Nt]  ulonglong2 {u_j, v_j}   64-bit fixed-point turns: u = frac(f_min t'_j), v = frac(df t'_j),
//                                        t'_j = t_j - t_0 (time origin shift, legal by eq. (2))
//   ws[B][nsplit][4][Nf] float           partial sums XC, XS, CC - n/2, CS of eq. (8) per time split
//   part_sum[B][nb], part_var[B][nb] double   block partials of sum x and sum (x - mean)^2
//   peak64[B] u64, counter[B] u32        packed arg-max and "last block" counters
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace lsp {

constexpr int TILE_Z = 256;               // samples staged in shared memory per tile of the FP32-pipe kernel
constexpr int MAX_PARTS = 128;            // max blocks per series in the pre-pass reductions

// 2 pi / 2^32: signed 32-bit phase (turns * 2^32) -> radians in [-pi, pi)
#define LSP_RAD_PER_PHASE 1.4629180792671596e-9f

typedef unsigned long long u64;

// ---- packed FP32 (f32x2) helpers: one instruction works on both lanes of a 64-bit register pair ----
__device__ __forceinline__ u64 pack2(float lo, float hi) {
    u64 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d;
}
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ u64 neg2(u64 a) {          // folded by ptxas into the consumer's operand negation
    float lo, hi; unpack2(a, lo, hi); return pack2(-lo, -hi);
}
__device__ __forceinline__ float sum2(u64 a) { float lo, hi; unpack2(a, lo, hi); return lo + hi; }

// ---- programmatic dependent launch (PDL): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor in the stream is still running; it must call pdl_wait() before it touches anything the predecessor
// writes (a no-op when launched normally).  pdl_trigger() in the predecessor lets the dependent grid be scheduled early.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- deterministic block reduction of a double (fixed shuffle tree, then fixed-order warp sums) ----
__device__ __forceinline__ double block_sum(double v, double* smem /* >= 32 doubles */) {
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) smem[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) { for (int i = 0; i < nw; ++i) r += smem[i]; smem[0] = r; }
    __syncthreads();
    r = smem[0];
    return r;
}

// frac(a*b) as 64-bit fixed-point turns, exact to ~2^-64 + the fp64 rounding of the operands:
// the product is split into its rounded value and the FMA residual so no bit of a*b is lost.
__device__ __forceinline__ u64 frac_fixed64(double a, double b, double* frac_out) {
    const double hi = a * b;
    const double lo = fma(a, b, -hi);
    double fr = hi - floor(hi);                                // exact, in [0,1] (1 only for tiny negative hi)
    if (!(fr < 1.0)) fr = 0.0;                                 // wrap: 1 == 0 (mod 1)
    u64 q = __double2ull_rz(fr * 18446744073709551616.0);      // exact: fr < 1 has <= 53 significant bits
    q += (u64)__double2ll_rn(lo * 18446744073709551616.0);     // |lo| <= 2^-53 |hi|: tiny, wraps mod 2^64
    if (frac_out) *frac_out = fr + lo;
    return q;
}

}  // namespace lsp
