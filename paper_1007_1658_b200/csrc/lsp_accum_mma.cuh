// lsp_accum_mma.cuh -- steps 3-5 of the hot path as a dense contraction on the tensor cores.
//
// The four sums of eq. (8) are, in complex form,
//     W(k) = XC + i XS          = sum_j X_j e^{i th_jk},         th_jk = 2 pi (f_min + k df) t_j
//     V(k) = (CC - SS) + 2i CS  = sum_j     e^{2 i th_jk}        (SS = Nt - CC)
// Split the frequency index k = kb + 32 h + l (l < 32).  The phase is then a SUM of a coarse and a
// fine part, th_jk = a_jh + b_jl with a_jh = 2 pi frac((f_min + (kb + 32 h) df) t_j) and
// b_jl = 2 pi frac(l df t_j), and e^{i(a+b)} = e^{ia} e^{ib} (angle addition) turns both sums into
// matrix products over the sample index j:
//     W[h,l] = sum_j (X_j e^{i a_jh}) (e^{i b_jl}),     V[h,l] = sum_j (e^{2i a_jh}) (e^{2i b_jl}).
// This is exact algebra (the same identity the rotation recurrence of lsp_accum*.cuh applies one
// step at a time); only (H + 32) trig values per sample are generated for H*32 frequencies, and the
// Nt*Nf multiply-adds of eq. (4) run as real 2x2-block GEMMs:
//     rows (h,C), (h,S);  K index (j,c), (j,s);  A[(h,C),(j,.)] = ( X cos a, -X sin a),
//     A[(h,S),(j,.)] = (X sin a, X cos a);  B[(j,c),l] = cos b, B[(j,s),l] = sin b.
//
// Precision: operands are fp16 hi + lo pairs (22 significant bits) and the product is formed as
// A_hi B_hi + A_lo B_hi + A_hi B_lo with fp32 accumulation (the dropped A_lo B_lo term is 2^-22);
// V needs only ~1e-3 relative accuracy of sqrt(Nt) against Nt and uses one fp16 pass.  X is scaled
// to unit variance first so fp16 neither overflows nor underflows.
// Register accumulators are folded into fp32 shared-memory sums every 1,024 samples (the chunked
// sums of PAPER.md:122), then written once per time split to `ws` -- no atomics, deterministic.
//
// Instruction: mma.sync.m16n8k16 (f16 in, f32 accumulate).  One warp owns 32 h x 32 l = 1,024
// frequencies: 4 x 4 MMA tiles, 2 x 64 fp32 accumulators per thread.  Each thread generates exactly the
// A-fragment elements it feeds (no shuffles): its row h = g (+8 mi) and its two samples tq, tq+4
// of the 8-sample k-step (g = lane/4, tq = lane%4).  The B fragments depend only on (j, l), are the
// same for all 8 warps of the CTA and are generated once per tile into shared memory.
#pragma once
#include "lsp_common.cuh"
#include "lsp_accum.cuh"
#include <cuda_fp16.h>

namespace lsp {

constexpr int REC_MMA = 4;
constexpr int MMA_WARPS = 8;                         // warps per CTA
constexpr int MMA_FPW = 1024;                        // frequencies per warp (32 h x 32 l)
constexpr int MMA_FPB = MMA_WARPS * MMA_FPW;         // frequencies per CTA
constexpr int MMA_TS = 128;                          // samples per shared-memory tile (16 k-steps)
constexpr int MMA_KSTEPS = MMA_TS / 8;
constexpr int MMA_FLUSH_TILES = 8;                   // fold every 1,024 samples
constexpr size_t MMA_SMEM = (size_t)MMA_TS * 16 + (size_t)MMA_KSTEPS * 6 * 32 * 16 + (size_t)128 * 256 * 4;

struct MmaParams {
    const float4* recA;
    const ulonglong2* recB;
    const double* part_var;     // [B][nparts]
    float* ws;                  // [B][nsplit][4][Nf]
    int64_t Nt, Nf;
    int64_t split_len;          // samples per split (multiple of MMA_TS)
    int nsplit, nfb, nparts;
    int unit_x;                 // 1: recA.x is a unit weight: no variance scaling
};

// 1 / sigma as the fp32 factor applied to X before it is split into fp16 pairs.  The finish kernel
// recomputes the identical value (same fixed-order sum, same IEEE operations) to undo it exactly.
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
__device__ __forceinline__ float2 unpack_h2(unsigned v)
{
    return __half22float2(*reinterpret_cast<const __half2*>(&v));
}
__device__ __forceinline__ void sincos_phase32(unsigned ph, float& c, float& s)
{
    const float ang = (float)(int)ph * LSP_RAD_PER_PHASE;      // signed 32-bit turns -> [-pi, pi)
    c = __cosf(ang); s = __sinf(ang);                            // MUFU, abs error ~2^-21
}
__device__ __forceinline__ void mma16816(float (&d)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3,
                                         unsigned b0, unsigned b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// grid.x = B * nsplit * nfb (frequency block fastest), 256 threads, MMA_SMEM bytes of dynamic shared memory.
__global__ void __launch_bounds__(MMA_WARPS * 32, 1) accum_mma_kernel(const MmaParams p)
{
    extern __shared__ uint4 lsp_smem_mma[];
    float4* rec = reinterpret_cast<float4*>(lsp_smem_mma);              // [TS] {X/sigma, pA32, wA32, 0}
    uint4* bfr = lsp_smem_mma + MMA_TS;                                 // [KSTEPS][hi,lo,V][ni pair][32 lanes] x {b0,b1,b0,b1}
    float* outer = reinterpret_cast<float*>(bfr + MMA_KSTEPS * 6 * 32); // [128][256]

    const unsigned tid = threadIdx.x, lane = tid & 31u, w = tid >> 5, g = lane >> 2, tq = lane & 3u;
    int64_t unit = blockIdx.x;
    const int fb = (int)(unit % p.nfb); unit /= p.nfb;
    const int sp = (int)(unit % p.nsplit);
    const int64_t b = unit / p.nsplit;
    const int64_t kb = (int64_t)fb * MMA_FPB;
    const int64_t j_begin = (int64_t)sp * p.split_len;
    const int64_t j_end = min(p.Nt, j_begin + p.split_len);
    const float4* recA = p.recA + b * p.Nt;
    const ulonglong2* recB = p.recB + b * p.Nt;
    const float xs = p.unit_x ? 1.f : x_scale(p.part_var + b * p.nparts, p.nparts, p.Nt);

    #pragma unroll 8
    for (int i = 0; i < 128; ++i) outer[i * 256 + tid] = 0.f;

    float acc[4][4][4], accD[4][4][4];                                  // [mi][ni][c]: W and V tiles
    #pragma unroll
    for (int mi = 0; mi < 4; ++mi)
        #pragma unroll
        for (int ni = 0; ni < 4; ++ni)
            #pragma unroll
            for (int c = 0; c < 4; ++c) { acc[mi][ni][c] = 0.f; accD[mi][ni][c] = 0.f; }

    const unsigned rowoff = 32u * w + g;                                // h of this thread's rows at mi = 0
    int tiles_since_flush = 0;

    for (int64_t j = j_begin; j < j_end; j += MMA_TS) {
        const int ns = (int)min((int64_t)MMA_TS, j_end - j);
        __syncthreads();                                                // previous tile fully consumed
        if (tid < MMA_TS) {
            float4 r = make_float4(0.f, 0.f, 0.f, 0.f);                 // pad: X = 0
            if ((int)tid < ns) {
                const float4 a = __ldg(recA + j + tid);
                const ulonglong2 q = __ldg(recB + j + tid);
                const u64 ph = q.x + (u64)kb * q.y;                     // u + kb v (mod 1, 64-bit wrap; reading G3)
                r.x = a.x * xs;
                r.y = __uint_as_float((unsigned)((ph + 0x80000000ull) >> 32));
                r.z = __uint_as_float((unsigned)((32ull * q.y + 0x80000000ull) >> 32));
            }
            rec[tid] = r;
        }
        // B fragments e^{i b_jl}, e^{2 i b_jl}: warp w fills k-steps w and w + 8, every thread the
        // register image its own lane will load (b0: sample tq, b1: sample tq + 4; column l = 8 ni + g).
        for (int s = (int)w; s < MMA_KSTEPS; s += MMA_WARPS) {
            unsigned q[3][4][2];                                        // [hi, lo, V][ni][b0, b1]
            #pragma unroll
            for (int half = 0; half < 2; ++half) {
                const int jj = 8 * s + 4 * half + (int)tq;
                const bool valid = jj < ns;
                const unsigned v32 = valid ? (unsigned)((__ldg(&recB[j + jj].y) + 0x80000000ull) >> 32) : 0u;
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni) {
                    float c, sn;
                    sincos_phase32((8u * ni + g) * v32, c, sn);
                    const unsigned hi = pack_h2(c, sn);
                    const float2 hf = unpack_h2(hi);
                    q[0][ni][half] = hi;
                    q[1][ni][half] = pack_h2(c - hf.x, sn - hf.y);
                    const float c2 = fmaf(c + c, c, -1.f), s2 = (c + c) * sn;
                    q[2][ni][half] = valid ? pack_h2(c2, s2) : 0u;      // pads must not count in V
                }
            }
            #pragma unroll
            for (int r = 0; r < 6; ++r) {                               // (b0, b1) of a column tile adjacent: MMA operand pairs
                const int kind = r >> 1, n0 = (r & 1) * 2;
                bfr[(s * 6 + r) * 32 + lane] = make_uint4(q[kind][n0][0], q[kind][n0][1], q[kind][n0 + 1][0], q[kind][n0 + 1][1]);
            }
        }
        __syncthreads();

        const int ksteps = (ns + 7) >> 3;
        #pragma unroll 1
        for (int s = 0; s < ksteps; ++s) {
            const float4 ra = rec[8 * s + tq];
            const float4 rb = rec[8 * s + 4 + tq];
            const uint4 bh01 = bfr[(s * 6 + 0) * 32 + lane], bh23 = bfr[(s * 6 + 1) * 32 + lane];
            const uint4 bl01 = bfr[(s * 6 + 2) * 32 + lane], bl23 = bfr[(s * 6 + 3) * 32 + lane];
            const uint4 bd01 = bfr[(s * 6 + 4) * 32 + lane], bd23 = bfr[(s * 6 + 5) * 32 + lane];
            const unsigned bh0[4] = {bh01.x, bh01.z, bh23.x, bh23.z}, bh1[4] = {bh01.y, bh01.w, bh23.y, bh23.w};
            const unsigned bl0[4] = {bl01.x, bl01.z, bl23.x, bl23.z}, bl1[4] = {bl01.y, bl01.w, bl23.y, bl23.w};
            const unsigned bd0[4] = {bd01.x, bd01.z, bd23.x, bd23.z}, bd1[4] = {bd01.y, bd01.w, bd23.y, bd23.w};
            const unsigned pa = __float_as_uint(ra.y), wa = __float_as_uint(ra.z);
            const unsigned pb = __float_as_uint(rb.y), wb = __float_as_uint(rb.z);
            #pragma unroll
            for (int mi = 0; mi < 4; ++mi) {
                // step 3: this thread's A elements, straight into fragment registers
                unsigned ah[4], al[4], ad[4];
                {
                    float c, sn;
                    sincos_phase32(pa + (rowoff + 8u * mi) * wa, c, sn);
                    const float xc = ra.x * c, xsn = ra.x * sn, nxsn = -ra.x * sn;
                    ah[0] = pack_h2(xc, nxsn);                          // row (h,C): ( X cos a, -X sin a)
                    ah[1] = pack_h2(xsn, xc);                           // row (h,S): ( X sin a,  X cos a)
                    const float2 h0 = unpack_h2(ah[0]);
                    const float rc = xc - h0.x, rs = xsn + h0.y, nrs = nxsn - h0.y;   // residuals of X cos a, +-X sin a
                    al[0] = pack_h2(rc, nrs);
                    al[1] = pack_h2(rs, rc);
                    const float cc = c + c, c2 = fmaf(cc, c, -1.f), s2 = cc * sn, ns2 = -cc * sn;
                    ad[0] = pack_h2(c2, ns2);
                    ad[1] = pack_h2(s2, c2);
                }
                {
                    float c, sn;
                    sincos_phase32(pb + (rowoff + 8u * mi) * wb, c, sn);
                    const float xc = rb.x * c, xsn = rb.x * sn, nxsn = -rb.x * sn;
                    ah[2] = pack_h2(xc, nxsn);
                    ah[3] = pack_h2(xsn, xc);
                    const float2 h0 = unpack_h2(ah[2]);
                    const float rc = xc - h0.x, rs = xsn + h0.y, nrs = nxsn - h0.y;
                    al[2] = pack_h2(rc, nrs);
                    al[3] = pack_h2(rs, rc);
                    const float cc = c + c, c2 = fmaf(cc, c, -1.f), s2 = cc * sn, ns2 = -cc * sn;
                    ad[2] = pack_h2(c2, ns2);
                    ad[3] = pack_h2(s2, c2);
                }
                // step 4: fragment order a0 = (row g, sample tq), a1 = (row g+8, sample tq),
                //         a2 = (row g, sample tq+4), a3 = (row g+8, sample tq+4)
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni) mma16816(acc[mi][ni], ah[0], ah[1], ah[2], ah[3], bh0[ni], bh1[ni]);
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni) mma16816(accD[mi][ni], ad[0], ad[1], ad[2], ad[3], bd0[ni], bd1[ni]);
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni) mma16816(acc[mi][ni], al[0], al[1], al[2], al[3], bh0[ni], bh1[ni]);
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni) mma16816(acc[mi][ni], ah[0], ah[1], ah[2], ah[3], bl0[ni], bl1[ni]);
            }
        }

        if (++tiles_since_flush == MMA_FLUSH_TILES || j + MMA_TS >= j_end) {
            // step 5: cascade
            #pragma unroll
            for (int mi = 0; mi < 4; ++mi)
                #pragma unroll
                for (int ni = 0; ni < 4; ++ni)
                    #pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const int i = (mi * 4 + ni) * 4 + c;
                        outer[i * 256 + tid] += acc[mi][ni][c];
                        outer[(64 + i) * 256 + tid] += accD[mi][ni][c];
                        acc[mi][ni][c] = 0.f; accD[mi][ni][c] = 0.f;
                    }
            tiles_since_flush = 0;
        }
    }

    // C fragment: c0,c1 = row g (h,C), columns 2 tq, 2 tq + 1;  c2,c3 = row g + 8 (h,S), same columns.
    float* ws = p.ws + ((b * p.nsplit + sp) * 4) * p.Nf;
    #pragma unroll
    for (int mi = 0; mi < 4; ++mi)
        #pragma unroll
        for (int ni = 0; ni < 4; ++ni)
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int64_t k = kb + (int64_t)(rowoff + 8u * mi) * 32 + 8 * ni + 2 * (int)tq + e;
                if (k < p.Nf) {
                    const int i = (mi * 4 + ni) * 4;
                    ws[0 * p.Nf + k] = outer[(i + e) * 256 + tid];                       // XC / sigma
                    ws[1 * p.Nf + k] = outer[(i + 2 + e) * 256 + tid];                   // XS / sigma
                    ws[2 * p.Nf + k] = 0.5f * outer[(64 + i + e) * 256 + tid];           // CC - n/2 = sum cos(2 th) / 2
                    ws[3 * p.Nf + k] = 0.5f * outer[(64 + i + 2 + e) * 256 + tid];       // CS       = sum sin(2 th) / 2
                }
            }
}

}  // namespace lsp
