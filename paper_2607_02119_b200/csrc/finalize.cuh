// K2 — top-k threshold, Gumbel-max over Philox4x32-10 noise, companion token sync and the
// delay-layout write (rows a3-a4 of DESIGN.md's hot-path table).
//
// One CTA per (request-owning batch row, stream).  The row's V temperature-scaled merged
// logits z (fp32, written by K1, normally still L2-resident) are turned into order-preserving
// 32-bit keys in shared memory; an exact 4-pass 8-bit radix select finds the k-th largest key
// (threshold semantics: every z >= threshold survives); only the survivors draw noise.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cfgms {

constexpr int kFinThreads = 256;

struct FinalizeParams {
    int R, S, V, NT;
    const float* z;           // [R][NT]
    const int32_t* pair_map;
    const float* temp;
    const int32_t* top_k;
    const int32_t* step;
    const uint32_t* req_id;   // nullable
    const int32_t* n_frames;  // nullable
    uint32_t seed_lo, seed_hi;
    int32_t pad_token;
    int32_t* tokens_out;      // [R][S]
    int32_t* delayed;         // nullable [R][T_cap][S]
    int32_t T_cap;
};

// Philox4x32-10 (Salmon et al. 2011): ten rounds of two 32x32->64 multiplies with key bumps.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// Standard Gumbel of token v: p = ((x >> 9) + 0.5) 2^-23 in (0,1) exactly representable in
// fp32; g = -ln(-ln(1 - p)) with log1p so the large-g tail (small p), which decides winners,
// keeps full relative accuracy.
__device__ __forceinline__ float gumbel_noise(uint32_t seed_lo, uint32_t seed_hi, uint32_t req, int tau, int stream,
                                              int v) {
    const uint4 o = philox4x32_10(make_uint4(static_cast<uint32_t>(v) >> 2, static_cast<uint32_t>(tau),
                                             static_cast<uint32_t>(stream), req),
                                  make_uint2(seed_lo, seed_hi));
    const int wsel = v & 3;
    const uint32_t x = wsel == 0 ? o.x : wsel == 1 ? o.y : wsel == 2 ? o.z : o.w;
    const float p = (static_cast<float>(x >> 9) + 0.5f) * 1.1920928955078125e-07f;  // 2^-23
    return -logf(-log1pf(-p));
}

__device__ __forceinline__ uint32_t float_key(float f) {
    f += 0.0f;  // -0 -> +0 so that equal floats have equal keys
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

__global__ void __launch_bounds__(kFinThreads) cfgms_finalize_kernel(const FinalizeParams p) {
    extern __shared__ uint32_t keys[];  // [V]
    __shared__ int hist[256];
    __shared__ uint32_t sel_prefix;
    __shared__ int sel_k;
    __shared__ float red_s[kFinThreads / 32];
    __shared__ int red_v[kFinThreads / 32];

    const int i = blockIdx.x;   // stream
    const int r = blockIdx.y;   // batch row
    const int tid = threadIdx.x;
    const int pm = p.pair_map[r];
    if (pm >= 0 && (r & 1)) return;  // companion row: its cond row writes both

    const int tau = p.step[r];
    const bool active = (i <= tau) && (p.n_frames == nullptr || tau - i < p.n_frames[r]);
    int token = p.pad_token;

    if (active) {
        const int V = p.V;
        const float* zr = p.z + static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * V;
        for (int v = tid; v < V; v += kFinThreads) keys[v] = float_key(zr[v]);
        __syncthreads();

        const float temp = p.temp[r];
        const int tk = p.top_k[r];
        const bool greedy = (tk == 1) || (temp == 0.f);
        uint32_t thr_key = 0u;
        if (!greedy && tk > 0 && tk < V) {
            // exact k-th largest key: MSB-first radix select, 8 bits per pass
            uint32_t prefix = 0u, mask = 0u;
            int k_rem = tk;
            for (int shift = 24; shift >= 0; shift -= 8) {
                hist[tid] = 0;   // kFinThreads == 256 bins
                __syncthreads();
                for (int v = tid; v < V; v += kFinThreads) {
                    const uint32_t key = keys[v];
                    if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1);
                }
                __syncthreads();
                if (tid < 32) {
                    // lane l owns digits [8l, 8l+8); suffix sums over higher digits
                    int cnt[8];
                    int sum = 0;
#pragma unroll
                    for (int j = 0; j < 8; ++j) { cnt[j] = hist[tid * 8 + j]; sum += cnt[j]; }
                    int above = 0;  // elements in lanes with higher digits
                    int incl = sum;
#pragma unroll
                    for (int off = 1; off < 32; off <<= 1) {
                        const int t = __shfl_down_sync(0xffffffffu, incl, off);
                        if (tid + off < 32) incl += t;
                    }
                    above = incl - sum;
                    // the k-th largest lies in this lane's digit range iff above < k_rem <= above + sum
                    if (above < k_rem && k_rem <= above + sum) {
                        int a = above;
#pragma unroll
                        for (int j = 7; j >= 0; --j) {
                            if (a < k_rem && k_rem <= a + cnt[j]) {
                                sel_prefix = prefix | (static_cast<uint32_t>(tid * 8 + j) << shift);
                                sel_k = k_rem - a;
                                break;
                            }
                            a += cnt[j];
                        }
                    }
                }
                __syncthreads();
                prefix = sel_prefix;
                k_rem = sel_k;
                mask |= 0xffu << shift;
                __syncthreads();
            }
            thr_key = prefix;
        }

        // argmax over survivors of s = z + g (or of z when greedy); lowest index wins ties
        float best_s = -INFINITY;
        int best_v = 0x7fffffff;
        const uint32_t req = p.req_id ? p.req_id[r] : static_cast<uint32_t>(r);
        for (int v = tid; v < V; v += kFinThreads) {
            const uint32_t key = keys[v];
            if (key >= thr_key) {
                float s = key_float(key);
                if (!greedy) s += gumbel_noise(p.seed_lo, p.seed_hi, req, tau, i, v);
                if (s > best_s || (s == best_s && v < best_v)) { best_s = s; best_v = v; }
            }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const float os = __shfl_xor_sync(0xffffffffu, best_s, off);
            const int ov = __shfl_xor_sync(0xffffffffu, best_v, off);
            if (os > best_s || (os == best_s && ov < best_v)) { best_s = os; best_v = ov; }
        }
        if ((tid & 31) == 0) { red_s[tid >> 5] = best_s; red_v[tid >> 5] = best_v; }
        __syncthreads();
        if (tid == 0) {
            for (int wi = 1; wi < kFinThreads / 32; ++wi) {
                const float os = red_s[wi];
                const int ov = red_v[wi];
                if (os > best_s || (os == best_s && ov < best_v)) { best_s = os; best_v = ov; }
            }
            token = best_v;
        }
    }
    if (tid == 0) {
        p.tokens_out[static_cast<size_t>(r) * p.S + i] = token;
        if (pm >= 0) p.tokens_out[static_cast<size_t>(pm) * p.S + i] = token;
        if (p.delayed) {
            const int slot = tau % p.T_cap;
            p.delayed[(static_cast<size_t>(r) * p.T_cap + slot) * p.S + i] = token;
        }
    }
}

}  // namespace cfgms
