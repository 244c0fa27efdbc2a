// K3 de-interleave, K4 bias fold, K5 fp32->bf16 cast.  All bandwidth-bound element kernels:
// coalesced 128-bit accesses, shared-memory staging only where the access pattern needs it.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace cfgms {

// ---------------------------------------------------------------- K3
// grid[q][f][i] = delayed[q][f + i][i].  One CTA turns frames [f0, f0 + kDeintFrames) of one
// request: it stages delayed rows [f0, f0 + kDeintFrames + S - 1) in shared memory with
// coalesced (128-bit when S % 4 == 0) loads, then writes the grid rows coalesced; the diagonal
// gather happens in shared memory (row stride S, column offset i: stride S + 1 words, which is
// bank-conflict free for even S).
constexpr int kDeintFrames = 256;
constexpr int kDeintThreads = 256;

__global__ void __launch_bounds__(kDeintThreads)
cfgms_deinterleave_kernel(const int32_t* __restrict__ delayed, int32_t* __restrict__ grid, int T, int S) {
    extern __shared__ int32_t tile[];  // [(kDeintFrames + S - 1) * S]
    const int F = T - S + 1;
    const int q = blockIdx.y;
    const int f0 = blockIdx.x * kDeintFrames;
    const int nf = min(kDeintFrames, F - f0);
    const int rows_in = nf + S - 1;
    const int32_t* src = delayed + (static_cast<size_t>(q) * T + f0) * S;
    int32_t* dst = grid + (static_cast<size_t>(q) * F + f0) * S;
    const int n_in = rows_in * S;
    const int n_out = nf * S;
    if ((S & 3) == 0) {
        // both bases are 16-byte aligned: (q*T + f0)*S and (q*F + f0)*S are multiples of 4 words
        const int4* src4 = reinterpret_cast<const int4*>(src);
        int4* tile4 = reinterpret_cast<int4*>(tile);
        for (int e = threadIdx.x; e < n_in / 4; e += kDeintThreads) tile4[e] = __ldg(src4 + e);
        __syncthreads();
        int4* dst4 = reinterpret_cast<int4*>(dst);
        const int s4 = S >> 2;
        for (int e = threadIdx.x; e < n_out / 4; e += kDeintThreads) {
            const int f = e / s4, i = (e - f * s4) * 4;
            int4 o;
            o.x = tile[(f + i) * S + i];
            o.y = tile[(f + i + 1) * S + i + 1];
            o.z = tile[(f + i + 2) * S + i + 2];
            o.w = tile[(f + i + 3) * S + i + 3];
            dst4[e] = o;
        }
    } else {
        for (int e = threadIdx.x; e < n_in; e += kDeintThreads) tile[e] = __ldg(src + e);
        __syncthreads();
        for (int e = threadIdx.x; e < n_out; e += kDeintThreads) {
            const int f = e / S, i = e - f * S;
            dst[e] = tile[(f + i) * S + i];
        }
    }
}

// ---------------------------------------------------------------- K4
// bias[i][v] = sum_k W_i[v][k] * e_i[k]: linearity of W_H (h_t + e_i) lets the stream embedding
// leave the per-step contraction.  One warp per output, fp64 accumulation (runs once).
__global__ void __launch_bounds__(256)
cfgms_bias_init_kernel(const __nv_bfloat16* __restrict__ heads, const __nv_bfloat16* __restrict__ embeds,
                       float* __restrict__ bias, int S, int V, int d) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const int NT = S * V;
    if (warp >= NT) return;
    const int i = warp / V;
    const __nv_bfloat16* wrow = heads + static_cast<size_t>(warp) * d;
    const __nv_bfloat16* e = embeds + static_cast<size_t>(i) * d;
    double acc = 0.0;
    for (int k = lane; k < d; k += 32)
        acc += static_cast<double>(__bfloat162float(wrow[k])) * static_cast<double>(__bfloat162float(e[k]));
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) bias[warp] = static_cast<float>(acc);
}

// ---------------------------------------------------------------- K5 (reading C18)
// fp32 hidden states -> bf16, round to nearest even.
__global__ void __launch_bounds__(256)
cfgms_cast_f32_bf16_kernel(const float* __restrict__ in, __nv_bfloat16* __restrict__ out, size_t n) {
    const size_t stride = static_cast<size_t>(gridDim.x) * blockDim.x;
    const size_t n4 = n / 4;
    const float4* in4 = reinterpret_cast<const float4*>(in);
    for (size_t e = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x; e < n4; e += stride) {
        const float4 v = __ldg(in4 + e);
        __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y);
        __nv_bfloat162 hi = __floats2bfloat162_rn(v.z, v.w);
        uint2 o;
        o.x = *reinterpret_cast<uint32_t*>(&lo);
        o.y = *reinterpret_cast<uint32_t*>(&hi);
        reinterpret_cast<uint2*>(out)[e] = o;
    }
    for (size_t e = n4 * 4 + static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x; e < n; e += stride)
        out[e] = __float2bfloat16_rn(in[e]);
}

// ---------------------------------------------------------------- K6 (PAPER.md:70-76 masking hook)
// bias[n] = base[n] + user[n]: the caller's additive vocabulary mask / bias is folded into the
// per-token bias the head GEMM's epilogue adds anyway.  user == nullptr restores the base.
__global__ void __launch_bounds__(256)
cfgms_bias_fold_kernel(const float* __restrict__ base, const float* __restrict__ user, float* __restrict__ bias, int n) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n) bias[e] = user ? base[e] + user[e] : base[e];
}

// Same fold with ragged per-stream vocabularies (one SSL stream + eight codec streams of
// different sizes on the uniform [S][V][d] layout): tokens v >= sizes[i] of stream i are masked with -inf.
struct StreamSizes {
    int32_t v[64];
};
__global__ void __launch_bounds__(256)
cfgms_bias_fold_ragged_kernel(const float* __restrict__ base, const float* __restrict__ user, float* __restrict__ bias,
                              int n, int V, const StreamSizes sizes) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int i = e / V, v = e - i * V;
    const float b = user ? base[e] + user[e] : base[e];
    bias[e] = v < sizes.v[i] ? b : -INFINITY;
}

// ---------------------------------------------------------------- K7 (PAPER.md:56 feedback)
// x[r][:] = bf16( sum_i emb[i][tokens[r][i]][:] ), fp32 accumulation in stream order.  One CTA per
// two-row slot; every thread owns 16-byte (8 x bf16) column chunks and keeps up to kFbUnroll
// independent gathers in flight.  When both rows of the slot carry the same tokens (a CFG pair
// after the token sync) the sum is formed once and stored twice.  HBM-bound:
// 2 * S * d bytes gathered per distinct row + 2 * d bytes written per row.
constexpr int kFbThreads = 256;
constexpr int kFbUnroll = 8;

__device__ __forceinline__ void fb_accumulate(float (&acc)[8], const uint4 v) {
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float2 f = __bfloat1622float2(h[q]);
        acc[2 * q] += f.x;
        acc[2 * q + 1] += f.y;
    }
}

__global__ void __launch_bounds__(kFbThreads)
cfgms_feedback_kernel(const int32_t* __restrict__ tokens, const __nv_bfloat16* __restrict__ emb,
                      __nv_bfloat16* __restrict__ x, int R, int S, int V_e, int d) {
    __shared__ int tok[2][64];
    __shared__ int same_s;
    const int r0 = 2 * blockIdx.x;
    const int rows = min(2, R - r0);
    if (threadIdx.x < 2 * S) {
        const int rr = threadIdx.x / S, i = threadIdx.x - rr * S;
        tok[rr][i] = rr < rows ? tokens[static_cast<size_t>(r0 + rr) * S + i] : -1;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int same = rows == 2;
        for (int i = 0; i < S; ++i) same &= tok[0][i] == tok[1][i];
        same_s = same;
    }
    __syncthreads();
    const bool same = same_s != 0;
    const int chunks = d >> 3;
    for (int rr = 0; rr < (same ? 1 : rows); ++rr) {
        for (int c = threadIdx.x; c < chunks; c += kFbThreads) {
            float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            for (int i0 = 0; i0 < S; i0 += kFbUnroll) {
                uint4 v[kFbUnroll];
#pragma unroll
                for (int u = 0; u < kFbUnroll; ++u) {
                    const int i = i0 + u;
                    const int t = i < S ? tok[rr][i] : -1;
                    v[u] = (t >= 0 && t < V_e)
                               ? __ldg(reinterpret_cast<const uint4*>(emb + (static_cast<size_t>(i) * V_e + t) * d) + c)
                               : make_uint4(0u, 0u, 0u, 0u);      // bf16 +0: contributes nothing
                }
#pragma unroll
                for (int u = 0; u < kFbUnroll; ++u) fb_accumulate(acc, v[u]);
            }
            uint4 o;
            __nv_bfloat162* oh = reinterpret_cast<__nv_bfloat162*>(&o);
#pragma unroll
            for (int q = 0; q < 4; ++q) oh[q] = __floats2bfloat162_rn(acc[2 * q], acc[2 * q + 1]);
            reinterpret_cast<uint4*>(x + static_cast<size_t>(r0 + rr) * d)[c] = o;
            if (same) reinterpret_cast<uint4*>(x + static_cast<size_t>(r0 + 1) * d)[c] = o;
        }
    }
}

}  // namespace cfgms
