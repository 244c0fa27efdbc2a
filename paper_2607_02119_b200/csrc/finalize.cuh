// K2 — top-k threshold, Gumbel-max over Philox4x32-10 noise, companion token sync and the
// delay-layout write (rows a3-a4 of DESIGN.md's hot-path table).
//
// Two samplers with identical semantics (readings C8-C12):
//
//  * cfgms_finalize_cand_kernel (the hot path: V % 32 == 0, V <= 8192) — ONE WARP per
//    (request-owning row, stream) cell, working on the V/8 values K1's epilogue emitted (top-4 of every
//    32-token chunk) instead of all V logits; chunks that may hide a top-k member are re-read from the
//    z spill.  Described in full above the kernel, further down in this file.
//
//  * cfgms_finalize_kernel<EPT> / cfgms_finalize_large_kernel (every other shape, and
//    CFGMS_CFG_NO_CANDIDATES) — one CTA of 256 threads per cell.  The row's V temperature-scaled
//    merged logits z (fp32, written by K1, normally still L2-resident) are loaded ONCE into registers
//    as order-preserving 32-bit keys.  Exact top-k threshold without sorting V values:
//      1. every thread takes the max of its V/256 keys; every warp extracts the ceil(k/8)-th
//         largest of its 32 thread maxima (redux.sync loop).  The minimum L of the 8 warp values
//         is a LOWER BOUND of the k-th largest key (at least 8*ceil(k/8) >= k keys are >= L);
//      2. keys >= L are compacted to shared memory (about 2k candidates in practice);
//      3. one warp runs an exact MSB-first 8-bit radix select on the candidates only;
//      4. survivors (key >= threshold; ties kept) draw Gumbel noise; block argmax, lowest index
//         on ties.
//    k > 256 (or V tiny) degrades gracefully: L = 0 and every key is a candidate.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx_sm100.cuh"

namespace cfgms {

constexpr int kFinThreads = 256;
constexpr int kFinWarps = kFinThreads / 32;

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
    const float* cand_val;    // [R][NT/32][4]  (candidate path only)
    const uint32_t* cand_src; // [R][NT/32]
    // Overlap with K1 (candidate path, V % 128 == 0): K1's epilogue warps count finished tiles per
    // (stream, row block) in ready[]; a cell is consumed once its group reached ready_target.
    // widenings (all nullable): forced tokens, streaming frame emission (include/cfgms.h)
    const int32_t* force_token;  // [R][S]
    int32_t* frame_out;          // [R][S]
    int32_t* frame_index_out;    // [R]
    int32_t eos_token;           // device-resident request state (include/cfgms.h): end-of-audio id, < 0 = none
    int32_t* step_next_out;      // [R]
    int32_t* n_frames_next_out;  // [R]
    int32_t* done_out;           // [R]
    int* ready;               // nullable [S][num_row_blocks]
    int* done;                // CTAs of this grid that finished; the last one clears ready[] for the next step
    unsigned long long* stats;// [16] cells that arrived before their group was complete (summed on the host)
    int* err;                 // sticky error word
    int BN, num_row_blocks, ready_target;
    // host-computed reciprocals (fast_div): x / d == (x * magic) >> 40 exactly for x * d < 2^40
    unsigned long long magic_per_stream;   // d = 2 * ceil(R / 2): cells per stream
    unsigned long long magic_bn;           // d = BN
    int poll_ns;              // sleep between two polls of a ready counter
    int pdl_wait;             // 1: launched as a programmatic dependent of K1 WITHOUT ready counters: the per-request
                              //    parameters are fetched while K1 still runs, then griddepcontrol.wait orders
                              //    everything K1 wrote (z, candidates) before the first read of it
    int stream_base, stream_stride;   // global stream of local stream i = base + i * stride (stream-sharded heads)
    int S_total;              // streams of the whole head (== S unless stream-sharded): ends the drain
    // per-request phase state machine (include/cfgms.h); phase == nullptr: plain path
    const int32_t* phase;        // [R]
    const int32_t* phase_pos;    // [R]
    int32_t* phase_next_out;     // [R] nullable
    int32_t* phase_pos_next_out; // [R] nullable
    int32_t* modality_out;       // [R] nullable
    // Stream-sharded heads (W5): the step's one exchange, an all-gather of the sampled
    // tokens, done by this kernel as direct stores into every rank's gather buffer (peer-mapped memory over
    // NVLink; this rank's own buffer included), followed by one flag per destination.  nullptr = off.
    int32_t* const* xchg_tokens; // device array [world] of int32 [2][xchg_rows][S_total] gather buffers (rank order);
                                 // the step that publishes epoch e writes half e & 1: a rank can run at most one
                                 // step ahead of a peer (its next step needs that peer's tokens), so the half it
                                 // overwrites has been consumed everywhere
    int xchg_half_elems;         // int32 elements between the two halves (same on every rank)
    uint32_t* const* xchg_flags; // device array [world] of uint32 [world] flag arrays: flags[q][rank] = epoch
    unsigned int* xchg_state;    // device, this rank's: [0] CTAs done (re-armed by the last one), [1] epoch published so far
    int xchg_world, xchg_rank;
    int V_text;                  // text region of stream 0: [0, V_text)
    int n_bridge;
    int32_t bridge[16];          // bridging tokens of the transition phase
#ifdef CFGMS_TRACE
    unsigned long long* trace;
#endif
};

// x / d for small non-negative x with magic = ceil(2^40 / d) (host: fast_div_magic): one wide multiply and a shift
// instead of the ~30-instruction division by a run-time value every cell would otherwise start with.
__host__ __device__ inline unsigned long long fast_div_magic(int d) { return ((1ull << 40) + static_cast<unsigned>(d) - 1) / static_cast<unsigned>(d); }
__device__ __forceinline__ int fast_div(int x, unsigned long long magic) {
    return static_cast<int>((static_cast<unsigned long long>(static_cast<unsigned>(x)) * magic) >> 40);
}

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
    // inner log1p keeps full relative accuracy of E = -ln(1-p) for small p; the outer logarithm may be
    // the fast one (abs. error <= 2^-21.4 near 1, <= 3 ulp elsewhere: < 1e-5 on |g| <= 17)
    return -__logf(-log1pf(-p));
}

// Order-preserving float -> uint32 (larger float <=> larger key).  Every real key is >= 1;
// 0 is reserved for "no element".
__device__ __forceinline__ uint32_t float_key(float f) {
    f += 0.0f;  // -0 -> +0 so that equal floats have equal keys
    const uint32_t u = __float_as_uint(f);
    const uint32_t k = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
    return k == 0u ? 1u : k;   // only the all-ones negative NaN maps to 0
}
__device__ __forceinline__ float key_float(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// Key of a value that is already canonical (K1 stores z + 0.0f) and not NaN: two instructions.
__device__ __forceinline__ uint32_t float_key_fast(float f) {
    const uint32_t u = __float_as_uint(f);
    return u ^ (static_cast<uint32_t>(static_cast<int32_t>(u) >> 31) | 0x80000000u);
}

// Stream-sharded heads (W5): this context may hold only the streams
// {base + i * stride}; the delay pattern, the noise key and the primary-stream rules use the GLOBAL index.
__device__ __forceinline__ int global_stream(const FinalizeParams& p, int i) { return p.stream_base + i * p.stream_stride; }

// Token of an ACTIVE cell given by the caller (phase machine hook), or -1.
__device__ __forceinline__ int forced_token(const FinalizeParams& p, int r, int i) {
    return p.force_token ? p.force_token[static_cast<size_t>(r) * p.S + i] : -1;
}

// What one (request, stream) cell does at this step.  Plain path (p.phase == nullptr): the request is in the
// audio phase with audio-local step tau_a = step[r].  With the phase state machine (include/cfgms.h):
//   TEXT        stream 0 samples from the text region [0, V_text), the other streams pad; want_modality
//   TRANSITION  stream 0 emits bridge[pos], the other streams pad
//   AUDIO       delay pattern on tau_a = pos; stream 0 samples from its audio region [V_text, V)
//   DONE        pad
constexpr int kPhaseText = 0, kPhaseTransition = 1, kPhaseAudio = 2, kPhaseDone = 3;
struct CellPlan {
    int phase;          // kPhaseAudio on the plain path
    int pos;            // phase_pos (== tau_a in the audio phase)
    int gstep;          // step[r]: keys the noise
    int tau_a;          // audio-local step (delay pattern, ring slot, frames); meaningful in the audio phase
    int lo, hi;         // vocabulary region the cell samples from
    int token;          // what an inactive cell emits (pad or a bridging token)
    bool sample;        // the cell draws a token from [lo, hi)
    bool want_modality; // TEXT phase, stream 0: also find the region of the unmasked argmax
};
__device__ __forceinline__ CellPlan plan_cell(const FinalizeParams& p, int r, int gi, int gstep, int F_req) {
    CellPlan c;
    c.phase = kPhaseAudio; c.pos = gstep; c.gstep = gstep; c.tau_a = gstep;
    c.lo = 0; c.hi = p.V; c.token = p.pad_token; c.sample = false; c.want_modality = false;
    if (p.phase) {
        c.phase = __ldcg(p.phase + r);
        c.pos = __ldcg(p.phase_pos + r);
        c.tau_a = c.pos;
    }
    if (c.phase == kPhaseAudio) {
        c.sample = (gi <= c.tau_a) && (c.tau_a - gi < F_req);
        if (p.phase && gi == 0) c.lo = p.V_text;
    } else if (c.phase == kPhaseText) {
        if (gi == 0) { c.sample = true; c.want_modality = true; c.hi = p.V_text; }
    } else if (c.phase == kPhaseTransition) {
        if (gi == 0 && c.pos >= 0 && c.pos < p.n_bridge) c.token = p.bridge[c.pos];
    }
    if (c.hi <= c.lo) c.sample = false;        // empty region: nothing to sample, the cell pads
    return c;
}
// TEXT phase with an EMPTY text region (V_text == 0: no phase table installed, or one without text tokens): the cell
// pads and reads no logits, but the modality inference still has an answer — every token of stream 0 is an audio token,
// so the unmasked argmax lies in the audio region whatever the logits are (the oracle computes it and gets 1).
__device__ __forceinline__ int modality_without_logits(const CellPlan& c) { return (c.want_modality && !c.sample) ? 1 : 0; }

// Rows a4 of the hot path, by ONE thread per cell: token to the row and its companion
// (PAPER.md:93), delayed-layout cell.  The thread of the LAST stream also emits
// the frame that completes at this step: f = tau - S + 1, frame[i] = ring[(f + i) mod
// T_cap][i]; streams i < S - 1 were written by earlier steps' launches, stream S - 1 is `token`.
// The thread of the PRIMARY stream's cell advances the request's state (phase, position, frame count).
__device__ __forceinline__ void write_cell(const FinalizeParams& p, int r, int i, int pm, const CellPlan& cp, int token,
                                           int modality) {
    const int tau = cp.tau_a;
    const bool audio = cp.phase == kPhaseAudio;
    p.tokens_out[static_cast<size_t>(r) * p.S + i] = token;
    if (pm >= 0) p.tokens_out[static_cast<size_t>(pm) * p.S + i] = token;
    if (p.xchg_tokens) {
        // all-gather by peer stores: cell [row][GLOBAL stream] of every rank's gather buffer
        const int gs = global_stream(p, i);
        const size_t half = ((__ldcg(p.xchg_state + 1) + 1u) & 1u) * static_cast<size_t>(p.xchg_half_elems);
        for (int q = 0; q < p.xchg_world; ++q) {
            int32_t* dst = p.xchg_tokens[q] + half;
            dst[static_cast<size_t>(r) * p.S_total + gs] = token;
            if (pm >= 0) dst[static_cast<size_t>(pm) * p.S_total + gs] = token;
        }
        __threadfence_system();        // ordered before this CTA's arrival below
    }
    if (p.delayed && audio) {          // only audio-phase tokens belong to the codebook matrix
        // ring slot tau mod T_cap (non-negative); a ring as deep as the request's lifetime needs no division at all
        const int slot = (tau >= 0 && tau < p.T_cap) ? tau : ((tau % p.T_cap) + p.T_cap) % p.T_cap;
        p.delayed[(static_cast<size_t>(r) * p.T_cap + slot) * p.S + i] = token;
    }
    if (global_stream(p, i) == 0) {
        // request state for the next step, by the thread of the PRIMARY stream's cell: the
        // frame count is fixed the moment stream 0 emits the end-of-audio token; other streams of this
        // step are unaffected (tau < tau + i), so nothing in this launch depends on what is written here
        constexpr int kUnset = 2147483647;
        int F = p.n_frames ? __ldcg(p.n_frames + r) : kUnset;
        int phase_next = cp.phase, pos_next = cp.pos;
        if (cp.phase == kPhaseText) {
            pos_next = 0;
            if (modality) phase_next = p.n_bridge > 0 ? kPhaseTransition : kPhaseAudio;
        } else if (cp.phase == kPhaseTransition) {
            if (cp.pos + 1 >= p.n_bridge) { phase_next = kPhaseAudio; pos_next = 0; }
            else pos_next = cp.pos + 1;
        } else if (audio) {
            if (F == kUnset && p.eos_token >= 0 && token == p.eos_token) F = tau;
            pos_next = tau + 1;
            if (F != kUnset && tau + 1 >= F + p.S_total - 1) phase_next = kPhaseDone;
        }
        if (p.step_next_out) p.step_next_out[r] = cp.gstep + 1;
        if (p.n_frames_next_out) p.n_frames_next_out[r] = F;
        if (p.done_out) p.done_out[r] = phase_next == kPhaseDone ? 1 : 0;
        if (p.phase_next_out) p.phase_next_out[r] = phase_next;
        if (p.phase_pos_next_out) p.phase_pos_next_out[r] = pos_next;
        if (p.modality_out) p.modality_out[r] = modality;
    }
    if (i == p.S - 1 && (p.frame_out || p.frame_index_out)) {
        const int f = tau - p.S + 1;
        const bool done = audio && f >= 0 && (p.n_frames == nullptr || f < __ldcg(p.n_frames + r)) && p.delayed && p.T_cap >= p.S;
        if (p.frame_index_out) {
            p.frame_index_out[r] = done ? f : -1;
            if (pm >= 0) p.frame_index_out[pm] = -1;
        }
        if (p.frame_out) {
            int32_t* fr = p.frame_out + static_cast<size_t>(r) * p.S;
            const int32_t* ring = p.delayed + static_cast<size_t>(r) * p.T_cap * p.S;
            for (int j = 0; j < p.S; ++j)
                fr[j] = !done ? p.pad_token : j == p.S - 1 ? token : __ldcg(ring + static_cast<size_t>((f + j) % p.T_cap) * p.S + j);
            if (pm >= 0)
                for (int j = 0; j < p.S; ++j) p.frame_out[static_cast<size_t>(pm) * p.S + j] = p.pad_token;
        }
    }
}

struct BestSV {
    float s;
    int v;
};
__device__ __forceinline__ void best_update(BestSV& b, float s, int v) {
    if (s > b.s || (s == b.s && v < b.v)) { b.s = s; b.v = v; }
}
// Block-wide argmax (lowest index on ties); result valid in thread 0.
__device__ __forceinline__ BestSV block_argmax(BestSV b, float* red_s, int* red_v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const float os = __shfl_xor_sync(0xffffffffu, b.s, off);
        const int ov = __shfl_xor_sync(0xffffffffu, b.v, off);
        best_update(b, os, ov);
    }
    const int tid = threadIdx.x;
    if ((tid & 31) == 0) { red_s[tid >> 5] = b.s; red_v[tid >> 5] = b.v; }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int wi = 1; wi < kFinWarps; ++wi) best_update(b, red_s[wi], red_v[wi]);
    }
    return b;
}

// Stream-sharded token exchange, end of the finalize grid (every thread of every CTA calls it): once all CTAs
// have stored their tokens into the peers' gather buffers, the last CTA publishes this rank's next epoch in
// flags[q][rank] of every rank q.  A rank's consumers wait until all `world` flags reached their own epoch
// (cfgms_exchange_wait_kernel).  The epoch lives on the device, so a captured graph replays correctly.
__device__ __forceinline__ void xchg_finish(const FinalizeParams& p) {
    if (!p.xchg_tokens) return;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence_system();
        const unsigned int total = gridDim.x * gridDim.y * gridDim.z;
        if (atomicAdd(p.xchg_state, 1u) == total - 1u) {
            p.xchg_state[0] = 0u;
            const unsigned int epoch = p.xchg_state[1] + 1u;
            p.xchg_state[1] = epoch;
            __threadfence_system();
            for (int q = 0; q < p.xchg_world; ++q) {
                volatile uint32_t* f = p.xchg_flags[q] + p.xchg_rank;
                *f = epoch;
            }
        }
    }
}

// Waits (bounded) until every rank's tokens of the current step have landed in THIS rank's gather buffer —
// flags[q] >= this rank's own wait count — and then copies the step's half into `latest`, the buffer consumers
// read (so nothing outside this kernel needs to know the epoch: CUDA-graph replay stays correct).  One CTA.
__global__ void __launch_bounds__(256)
cfgms_exchange_wait_kernel(const volatile uint32_t* flags, unsigned int* wait_count, int world, const int32_t* halves,
                           int32_t* latest, int half_elems, int n_copy, int* err) {
    __shared__ unsigned int want;
    __shared__ int timed_out;
    if (threadIdx.x == 0) { want = *wait_count + 1u; timed_out = 0; }
    __syncthreads();
    if (static_cast<int>(threadIdx.x) < world) {
        const uint64_t t0 = global_timer_ns();
        while (static_cast<int>(flags[threadIdx.x] - want) < 0) {
            __nanosleep(200);
            if (global_timer_ns() - t0 > 2000000000ull) {
                // A late peer (first-step module load, a slow rank) must not poison this process's CUDA context: latch the
                // time-out in the sticky error word and leave.  `latest` and the wait count stay as they were, so the
                // step can be waited for again once cfgms_last_device_error has reported it.
                atomicCAS(err, 0, 7 /* CFGMS_ERR_TIMEOUT */ | (11 << 8));
                timed_out = 1;
                break;
            }
        }
    }
    __threadfence_system();      // acquire side
    __syncthreads();
    if (timed_out) return;
    const int32_t* src = halves + static_cast<size_t>(want & 1u) * half_elems;
    for (int e = threadIdx.x; e < n_copy; e += blockDim.x) latest[e] = __ldcv(src + e);
    if (threadIdx.x == 0) *wait_count = want;
}

// Exact k-th largest (1-based, with multiplicity) of n keys in shared memory, by ONE warp:
// MSB-first radix select, 8 bits per pass.  Requires 1 <= k <= n.
struct SmemKeys {
    const uint32_t* keys;
    __device__ __forceinline__ uint32_t operator()(int e) const { return keys[e]; }
};
template <class Load>
__device__ __forceinline__ uint32_t warp_radix_select(const Load load, int n, int k, int* hist, int lane) {
    uint32_t prefix = 0u, mask = 0u;
    for (int shift = 24; shift >= 0; shift -= 8) {
#pragma unroll
        for (int j = 0; j < 8; ++j) hist[lane * 8 + j] = 0;
        __syncwarp();
        for (int e = lane; e < n; e += 32) {
            const uint32_t key = load(e);
            if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1);
        }
        __syncwarp();
        int cnt[8];
        int sum = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) { cnt[j] = hist[lane * 8 + j]; sum += cnt[j]; }
        int incl = sum;  // inclusive suffix sum over lanes (higher lanes hold higher digits)
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int t = __shfl_down_sync(0xffffffffu, incl, off);
            if (lane + off < 32) incl += t;
        }
        const int above = incl - sum;
        uint32_t digit = 0;
        int k_next = 0;
        const bool mine = above < k && k <= above + sum;
        if (mine) {
            int a = above;
#pragma unroll
            for (int j = 7; j >= 0; --j) {
                if (a < k && k <= a + cnt[j]) { digit = static_cast<uint32_t>(lane * 8 + j); k_next = k - a; break; }
                a += cnt[j];
            }
        }
        const uint32_t owner = __ballot_sync(0xffffffffu, mine);
        const int src = __ffs(owner) - 1;
        digit = __shfl_sync(0xffffffffu, digit, src);
        k = __shfl_sync(0xffffffffu, k_next, src);
        prefix |= digit << shift;
        mask |= 0xffu << shift;
        __syncwarp();
    }
    return prefix;
}

// EPT = keys per thread held in registers; supports V <= 256 * EPT.
template <int EPT>
__global__ void __launch_bounds__(kFinThreads) cfgms_finalize_kernel(const FinalizeParams p) {
    extern __shared__ uint32_t dyn[];  // cand_key[V] | cand_idx[V]
    __shared__ int hist[256];
    __shared__ uint32_t warp_kth[kFinWarps];
    __shared__ int n_cand;
    __shared__ uint32_t thr_key_s;
    __shared__ float red_s[kFinWarps];
    __shared__ int red_v[kFinWarps];

    pdl_launch_dependents();    // the next kernel in the stream may be set up while this one runs
    const int i = blockIdx.x;   // stream
    const int r = blockIdx.y;   // batch row
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const int pm = p.pair_map[r];
    if (pm >= 0 && (r & 1)) { xchg_finish(p); return; }  // companion row: its cond row writes both

    const int gi = global_stream(p, i);
    const CellPlan cp = plan_cell(p, r, gi, __ldcg(p.step + r), p.n_frames ? __ldcg(p.n_frames + r) : 2147483647);
    const int tau = cp.gstep;          // keys the noise
    bool active = cp.sample;
    int token = cp.token;
    int modality = modality_without_logits(cp);
    if (active) {
        const int ft = forced_token(p, r, i);
        if (ft >= 0) { token = ft; active = false; }
    }

    if (active) {
        const int V = p.V;
        const int Vr = cp.hi - cp.lo;      // size of the vocabulary region this cell samples from
        uint32_t* cand_key = dyn;
        int* cand_idx = reinterpret_cast<int*>(dyn + V);
        const float* zr = p.z + static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * V;
        uint32_t key[EPT];
#pragma unroll
        for (int j = 0; j < EPT; ++j) {
            const int v = j * kFinThreads + tid;
            key[j] = v < V ? float_key(__ldg(zr + v)) : 0u;
        }
        if (cp.want_modality) {
            // the modality the model asks for: region of the argmax of the UNMASKED logits (lowest token on ties)
            BestSV m = {-INFINITY, 0x7fffffff};
#pragma unroll
            for (int j = 0; j < EPT; ++j)
                if (key[j] != 0u) best_update(m, key_float(key[j]), j * kFinThreads + tid);
            m = block_argmax(m, red_s, red_v);
            if (tid == 0) modality = m.v >= p.V_text ? 1 : 0;
            __syncthreads();               // red_s / red_v are reused by the sampling argmax below
        }
#pragma unroll
        for (int j = 0; j < EPT; ++j) {    // dynamic vocabulary masking: tokens outside the region do not exist
            const int v = j * kFinThreads + tid;
            if (v < cp.lo || v >= cp.hi) key[j] = 0u;
        }
        const float temp = p.temp[r];
        const int tk = p.top_k[r];
        const bool greedy = (tk == 1) || (temp == 0.f);
        const bool filter = !greedy && tk > 0 && tk < Vr;
        const uint32_t req = p.req_id ? p.req_id[r] : static_cast<uint32_t>(r);
        BestSV best = {-INFINITY, 0x7fffffff};

        if (filter) {
            if (tid == 0) n_cand = 0;
            // 1. lower bound L of the k-th largest key
            uint32_t m = 0u;
#pragma unroll
            for (int j = 0; j < EPT; ++j) m = max(m, key[j]);
            const int kp = (tk + kFinWarps - 1) / kFinWarps;
            uint32_t kth = 0u;
            if (kp <= 32) {
                uint32_t cur = m;
                for (int it = 0; it < kp; ++it) {
                    kth = __reduce_max_sync(0xffffffffu, cur);
                    const uint32_t who = __ballot_sync(0xffffffffu, cur == kth);
                    if (lane == __ffs(who) - 1) cur = 0u;
                }
            }
            if (lane == 0) warp_kth[warp] = kth;
            __syncthreads();
            uint32_t L = warp_kth[0];
#pragma unroll
            for (int wi = 1; wi < kFinWarps; ++wi) L = min(L, warp_kth[wi]);
            if (L == 0u) L = 1u;  // every real key
            // 2. compact candidates (key >= L)
#pragma unroll
            for (int j = 0; j < EPT; ++j) {
                const bool pred = key[j] >= L;
                const uint32_t b = __ballot_sync(0xffffffffu, pred);
                if (b) {
                    int base = 0;
                    if (lane == 0) base = atomicAdd(&n_cand, __popc(b));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (pred) {
                        const int pos = base + __popc(b & ((1u << lane) - 1u));
                        cand_key[pos] = key[j];
                        cand_idx[pos] = j * kFinThreads + tid;
                    }
                }
            }
            __syncthreads();
            const int C = n_cand;
            // 3. exact threshold among the candidates
            if (warp == 0) {
                const uint32_t t = warp_radix_select(SmemKeys{cand_key}, C, tk, hist, lane);
                if (lane == 0) thr_key_s = t;
            }
            __syncthreads();
            const uint32_t thr_key = thr_key_s;
            // 4. Gumbel-max over the survivors
            for (int e = tid; e < C; e += kFinThreads) {
                const uint32_t ck = cand_key[e];
                if (ck >= thr_key) {
                    const int v = cand_idx[e];
                    best_update(best, key_float(ck) + gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, v), v);
                }
            }
        } else {
            // greedy argmax, or no top-k filter: every token competes
#pragma unroll
            for (int j = 0; j < EPT; ++j) {
                const int v = j * kFinThreads + tid;
                if (key[j] != 0u) {
                    float s = key_float(key[j]);
                    if (!greedy) s += gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, v);
                    best_update(best, s, v);
                }
            }
        }
        best = block_argmax(best, red_s, red_v);
        token = best.v;
    }
    if (tid == 0) write_cell(p, r, i, pm, cp, token, modality);
    xchg_finish(p);
}

// Fallback for V > 256 * 32: keys in shared memory, radix select over all of them.
__global__ void __launch_bounds__(kFinThreads) cfgms_finalize_large_kernel(const FinalizeParams p) {
    extern __shared__ uint32_t dyn[];  // keys[V]
    __shared__ int hist[256];
    __shared__ uint32_t thr_key_s;
    __shared__ float red_s[kFinWarps];
    __shared__ int red_v[kFinWarps];

    pdl_launch_dependents();
    const int i = blockIdx.x, r = blockIdx.y, tid = threadIdx.x;
    const int pm = p.pair_map[r];
    if (pm >= 0 && (r & 1)) { xchg_finish(p); return; }
    const int gi = global_stream(p, i);
    const CellPlan cp = plan_cell(p, r, gi, __ldcg(p.step + r), p.n_frames ? __ldcg(p.n_frames + r) : 2147483647);
    const int tau = cp.gstep;          // keys the noise
    bool active = cp.sample;
    int token = cp.token;
    int modality = modality_without_logits(cp);
    if (active) {
        const int ft = forced_token(p, r, i);
        if (ft >= 0) { token = ft; active = false; }
    }
    if (active) {
        const int V = p.V;
        const int Vr = cp.hi - cp.lo;
        const float* zr = p.z + static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * V;
        for (int v = tid; v < V; v += kFinThreads) dyn[v] = float_key(__ldg(zr + v));
        __syncthreads();
        if (cp.want_modality) {            // region of the argmax of the unmasked logits
            BestSV m = {-INFINITY, 0x7fffffff};
            for (int v = tid; v < V; v += kFinThreads) best_update(m, key_float(dyn[v]), v);
            m = block_argmax(m, red_s, red_v);
            if (tid == 0) modality = m.v >= p.V_text ? 1 : 0;
            __syncthreads();
        }
        const float temp = p.temp[r];
        const int tk = p.top_k[r];
        const bool greedy = (tk == 1) || (temp == 0.f);
        uint32_t thr_key = 0u;
        if (!greedy && tk > 0 && tk < Vr) {
            if (tid < 32) {
                const uint32_t t = warp_radix_select(SmemKeys{dyn + cp.lo}, Vr, tk, hist, tid);
                if (tid == 0) thr_key_s = t;
            }
            __syncthreads();
            thr_key = thr_key_s;
        }
        const uint32_t req = p.req_id ? p.req_id[r] : static_cast<uint32_t>(r);
        BestSV best = {-INFINITY, 0x7fffffff};
        for (int v = cp.lo + tid; v < cp.hi; v += kFinThreads) {
            const uint32_t k = dyn[v];
            if (k >= thr_key) {
                float s = key_float(k);
                if (!greedy) s += gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, v);
                best_update(best, s, v);
            }
        }
        best = block_argmax(best, red_s, red_v);
        token = best.v;
    }
    if (tid == 0) write_cell(p, r, i, pm, cp, token, modality);
    xchg_finish(p);
}


// ---------------------------------------------------------------------------------------------
// Candidate path (V % 32 == 0, V <= 8192): ONE WARP per (request-owning row, stream) works on the
// V/8 values K1's epilogue emitted (top-4 of every 32-token chunk, descending) instead of all V
// logits.  Lane l keeps chunks l, l+32, ... in registers.
//   t_E = k-th largest emitted value  <=  true threshold (the emitted set is a subset);
//   K1 selects with 27-bit key buckets, so a value it did NOT emit has
//   float_key(hidden) <= float_key(smallest emitted) | 31: a chunk with (key4 | 31) < t_E cannot
//   hide anything >= t_E and its emitted values >= t_E are all of its candidates; a chunk whose
//   bound reaches t_E ("overflow") is re-read in full from the z spill.  The candidate set {z >= t_E} is then complete and the
//   exact threshold is its k-th largest (= t_E when no chunk overflowed).
// t_E itself: with j = ceil(k / G), lo = min over chunks of their j-th value is a lower bound
// (G*j >= k values are >= lo); ONE histogram pass with 256 linear buckets over [lo, max] finds
// the bucket of the k-th largest, and the few values of that bucket are ranked exactly.
// k > V/8 or no filter: the warp scans the full row from the spill (exact, slow, rare).
constexpr int kCandWarps = 4;

struct GlobalKeys {
    const float* z;
    __device__ __forceinline__ uint32_t operator()(int e) const { return float_key(__ldcg(z + e)); }
};

__device__ __forceinline__ BestSV warp_argmax(BestSV b) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const float os = __shfl_xor_sync(0xffffffffu, b.s, off);
        const int ov = __shfl_xor_sync(0xffffffffu, b.v, off);
        best_update(b, os, ov);
    }
    return b;
}

// per-warp shared memory (32-bit words): hist[256] | small[32] | misc[8] | list_key[cap] | list_v[cap]
__host__ __device__ constexpr int cand_list_cap(int V) { return V / 8 + 32; }
__host__ __device__ constexpr int cand_warp_words(int V) { return 256 + 32 + 8 + 2 * cand_list_cap(V); }

template <int CPL>   // chunks per lane: V <= 1024 * CPL
__global__ void __launch_bounds__(kCandWarps * 32) cfgms_finalize_cand_kernel(const FinalizeParams p) {
    extern __shared__ uint32_t dyn[];
    // The next kernel in the stream (normally the next step's head GEMM, launched as a programmatic
    // dependent) may be scheduled and set up while this grid runs; it waits for this grid's completion
    // (griddepcontrol.wait) before it touches anything this grid reads or writes.
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
#ifdef CFGMS_TRACE
    const bool tr = threadIdx.x == 0;
    if (tr) { CFGMS_TRACE_MARK(p.trace, 0); CFGMS_TRACE_MARK(p.trace, 1); }
#define CFGMS_K2_MARK(slot) do { if (tr) CFGMS_TRACE_MARK(p.trace, slot); } while (0)
#else
#define CFGMS_K2_MARK(slot) ((void)0)
#endif
    // Cells in the order K1 finishes them: stream-major; inside a stream first every EVEN row (ascending =
    // row blocks ascending), then every odd row.  Companion rows are odd rows, so in a CFG batch the warps
    // with nothing to do fill whole CTAs, which retire at once instead of holding resident CTAs half empty.
    const int slots = (p.R + 1) >> 1;
    const int per_stream = 2 * slots;
    const int cell = blockIdx.x * kCandWarps + warp;
    const bool in_grid = cell < per_stream * p.S;
    const int i = in_grid ? fast_div(cell, p.magic_per_stream) : 0;
    const int rem = in_grid ? cell - i * per_stream : 0;
    const int half = rem >= slots ? 1 : 0;
    const int r_raw = 2 * (rem - half * slots) + half;
    const bool in_range = in_grid && r_raw < p.R;
    const int r = in_range ? r_raw : 0;
    // every per-request parameter is requested here, before any of them is used: one L2 round trip for
    // all of them instead of one per dependent use (row r is always a readable row)
    // (step / n_frames may be the previous step's step_next_out / n_frames_next_out: read through L2)
    const int pm = p.pair_map[r];
    const int gstep = __ldcg(p.step + r);
    const int F_req = p.n_frames ? __ldcg(p.n_frames + r) : 2147483647;
    const int gi = global_stream(p, i);
    const CellPlan cp = plan_cell(p, r, gi, gstep, F_req);   // phase, vocabulary region, audio-local step
    const int tau = cp.gstep;                                 // keys the noise
    const float temp = p.temp[r];
    const int tk_raw = p.top_k[r];
    const uint32_t req = p.req_id ? p.req_id[r] : static_cast<uint32_t>(r);
    const int ft = forced_token(p, r, i);
    const bool valid = in_range && !(pm >= 0 && (r & 1));   // a companion row is written by its cond row
    // Serial mode, small grids: this grid was scheduled while the head GEMM was still running (programmatic
    // dependent launch); its launch latency and the parameter fetch above are behind it when the GEMM ends.
    if (p.pdl_wait) pdl_wait_primary();

    // The cell samples from the vocabulary region [cp.lo, cp.hi) of its stream (the whole sub-vocabulary on the
    // plain path; whole 32-token chunks always: the host checks the phase table).  Everything below works in
    // region-local tokens and chunks; `tok0` turns them back into tokens of the stream.
    const int tok0 = cp.lo;
    const int V = cp.hi - cp.lo;     // tokens of the region
    const int G = V >> 5;            // chunks of the region
    const int E = G * 4;             // emitted values
    const int cap = cand_list_cap(p.V);
    int* hist = reinterpret_cast<int*>(dyn + static_cast<size_t>(warp) * cand_warp_words(p.V));
    uint32_t* small = reinterpret_cast<uint32_t*>(hist + 256);
    int* misc = reinterpret_cast<int*>(small + 32);
    uint32_t* list_key = reinterpret_cast<uint32_t*>(misc + 8);
    int* list_v = reinterpret_cast<int*>(list_key + cap);

    bool active = valid && cp.sample;
    int token = cp.token;
    int modality = modality_without_logits(cp);
    if (active && ft >= 0) { token = ft; active = false; }
    if (valid && p.ready) {
        // Wait until K1 has written every tile of this (stream, row block): the acquire pairs with the
        // epilogue warps' red.release.  EVERY request-owning cell waits, also a PAD or forced one that
        // reads nothing: the last CTA of this grid re-arms the counters, which is only safe once
        // every group is complete, i.e. once K1 will not signal again.  Bounded: a pipeline bug fails loudly.
        const int* flag = p.ready + i * p.num_row_blocks + fast_div(r, p.magic_bn);
        if (lane == 0 && ld_acquire_gpu(flag) < p.ready_target) {
            atomicAdd(p.stats + (blockIdx.x & 15), 1ull);   // evidence counter, spread over 16 words
            const uint64_t t0 = global_timer_ns();
            while (ld_acquire_gpu(flag) < p.ready_target) {
                __nanosleep(p.poll_ns);
                if (global_timer_ns() - t0 > 2000000000ull) {
                    atomicCAS(p.err, 0, 7 /* CFGMS_ERR_TIMEOUT */ | (9 << 8));
                    __threadfence_system();
                    __trap();
                }
            }
        }
        __syncwarp();
    }
    CFGMS_K2_MARK(2);      // parameters in, readiness wait over
    if (active) {
        const float* zr = p.z + static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * p.V + tok0;
        const size_t chunk0 = (static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * p.V + tok0) >> 5;
        if (cp.want_modality) {
            // The modality the model asks for: region of the argmax of stream 0's UNMASKED logits.
            // Every chunk's first emitted value is its exact maximum (lowest token among equals), so the row's
            // argmax is the best of the chunk maxima — over ALL chunks of the stream, not only the region's.
            const size_t row0 = (static_cast<size_t>(r) * p.NT + static_cast<size_t>(i) * p.V) >> 5;
            BestSV m = {-INFINITY, 0x7fffffff};
            for (int c = lane; c < (p.V >> 5); c += 32) {
                const float top = __ldcg(p.cand_val + (row0 + c) * 4);
                const uint32_t off = __ldcg(p.cand_src + row0 + c) & 31u;
                best_update(m, top, c * 32 + static_cast<int>(off));
            }
            m = warp_argmax(m);
            modality = m.v >= p.V_text ? 1 : 0;
        }
        const bool greedy = (tk_raw == 1) || (temp == 0.f);
        const bool filter = !greedy && tk_raw > 0 && tk_raw < V;
        const int tk = greedy ? 1 : tk_raw;   // greedy = exact top-1 (ties: lowest token), no noise
        BestSV best = {-INFINITY, 0x7fffffff};

        if (greedy || (filter && tk <= E)) {
            uint32_t key[CPL][4];
            uint32_t src[CPL];
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                const int c = j * 32 + lane;
                if (c < G) {
                    const float4 v4 = __ldcg(reinterpret_cast<const float4*>(p.cand_val) + chunk0 + c);
                    src[j] = __ldcg(p.cand_src + chunk0 + c);
                    key[j][0] = float_key_fast(v4.x); key[j][1] = float_key_fast(v4.y);
                    key[j][2] = float_key_fast(v4.z); key[j][3] = float_key_fast(v4.w);
                } else {
                    src[j] = 0u;
                    key[j][0] = key[j][1] = key[j][2] = key[j][3] = 0u;
                }
            }
            CFGMS_K2_MARK(3);      // emitted values loaded
            {
                // ---- t_E: k-th largest of the E emitted values
                const int jj = (tk + G - 1) / G - 1;           // 0..3: the (jj+1)-th value of every chunk
                uint32_t lo = 0xffffffffu, hi = 0u;
#pragma unroll
                for (int j = 0; j < CPL; ++j) {
                    if (j * 32 + lane < G) {
                        const uint32_t kj = jj == 0 ? key[j][0] : jj == 1 ? key[j][1] : jj == 2 ? key[j][2] : key[j][3];
                        lo = min(lo, kj);
                        hi = max(hi, key[j][0]);
                    }
                }
                lo = __reduce_min_sync(0xffffffffu, lo);
                hi = __reduce_max_sync(0xffffffffu, hi);
                const uint32_t range = hi - lo;
                const int shift = range < 256u ? 0 : (24 - __clz(range));   // (key - lo) >> shift <= 255
#pragma unroll
                for (int j = 0; j < 8; ++j) hist[lane * 8 + j] = 0;
                if (lane == 0) misc[0] = 0;
                __syncwarp();
#pragma unroll
                for (int j = 0; j < CPL; ++j)
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        if (key[j][e] >= lo) atomicAdd(&hist[(key[j][e] - lo) >> shift], 1);
                __syncwarp();
                int cnt[8];
                int sum = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) { cnt[j] = hist[lane * 8 + j]; sum += cnt[j]; }
                int incl = sum;
#pragma unroll
                for (int off = 1; off < 32; off <<= 1) {
                    const int t = __shfl_down_sync(0xffffffffu, incl, off);
                    if (lane + off < 32) incl += t;
                }
                const int above = incl - sum;
                int bucket = 0, k_rem = 0, m_in = 0;
                const bool mine = above < tk && tk <= above + sum;
                if (mine) {
                    int a = above;
#pragma unroll
                    for (int j = 7; j >= 0; --j) {
                        if (a < tk && tk <= a + cnt[j]) { bucket = lane * 8 + j; k_rem = tk - a; m_in = cnt[j]; break; }
                        a += cnt[j];
                    }
                }
                const int owner = __ffs(__ballot_sync(0xffffffffu, mine)) - 1;
                bucket = __shfl_sync(0xffffffffu, bucket, owner);
                k_rem = __shfl_sync(0xffffffffu, k_rem, owner);
                m_in = __shfl_sync(0xffffffffu, m_in, owner);
                uint32_t tE = 0u;
                if (m_in <= 32) {
                    // rank the few values of that bucket exactly: every lane counts its members, one warp scan gives
                    // each lane its place in small[] (no atomics with a return value on the latency chain)
                    int mine_b = 0;
#pragma unroll
                    for (int j = 0; j < CPL; ++j)
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            mine_b += (key[j][e] >= lo && static_cast<int>((key[j][e] - lo) >> shift) == bucket) ? 1 : 0;
                    int at = mine_b;
#pragma unroll
                    for (int off = 1; off < 32; off <<= 1) {
                        const int t = __shfl_up_sync(0xffffffffu, at, off);
                        if (lane >= off) at += t;
                    }
                    at -= mine_b;
#pragma unroll
                    for (int j = 0; j < CPL; ++j)
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (key[j][e] >= lo && static_cast<int>((key[j][e] - lo) >> shift) == bucket) small[at++] = key[j][e];
                    __syncwarp();
                    const uint32_t x = lane < m_in ? small[lane] : 0u;
                    int gt = 0, ge = 0;
                    for (int q = 0; q < m_in; ++q) {
                        const uint32_t y = small[q];
                        gt += y > x;
                        ge += y >= x;
                    }
                    const bool hit = lane < m_in && gt < k_rem && k_rem <= ge;
                    const int who = __ffs(__ballot_sync(0xffffffffu, hit)) - 1;
                    tE = __shfl_sync(0xffffffffu, x, who);
                } else {
                    // many (near-)equal values in one bucket: generic radix select over all emitted values
#pragma unroll
                    for (int j = 0; j < CPL; ++j)
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (j * 32 + lane < G) list_key[(j * 32 + lane) * 4 + e < cap ? (j * 32 + lane) * 4 + e : 0] = key[j][e];
                    __syncwarp();
                    tE = E <= cap ? warp_radix_select(SmemKeys{list_key}, E, tk, hist, lane) : 0u;
                    __syncwarp();
                }
                CFGMS_K2_MARK(4);  // t_E known
                // ---- candidate list {z >= t_E}; overflowing chunks are re-read in full
                // (every lane counts its entries, one warp scan places them: one shuffle chain instead of a ballot per value)
                int n_list = 0;
                uint32_t any_overflow = 0u;
                {
                    int mine_l = 0;
                    bool my_ovf = false;
#pragma unroll
                    for (int j = 0; j < CPL; ++j) {
                        const int c = j * 32 + lane;
                        const bool ovf = c < G && (key[j][3] | 31u) >= tE;
                        my_ovf |= ovf;
#pragma unroll
                        for (int e = 0; e < 4; ++e) mine_l += (c < G && !ovf && key[j][e] >= tE) ? 1 : 0;
                    }
                    any_overflow = __ballot_sync(0xffffffffu, my_ovf);
                    int at = mine_l;
#pragma unroll
                    for (int off = 1; off < 32; off <<= 1) {
                        const int t = __shfl_up_sync(0xffffffffu, at, off);
                        if (lane >= off) at += t;
                    }
                    n_list = __shfl_sync(0xffffffffu, at, 31);
                    at -= mine_l;
#pragma unroll
                    for (int j = 0; j < CPL; ++j) {
                        const int c = j * 32 + lane;
                        const bool ovf = c < G && (key[j][3] | 31u) >= tE;
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            if (c < G && !ovf && key[j][e] >= tE) {
                                list_key[at] = key[j][e];
                                list_v[at] = tok0 + c * 32 + static_cast<int>((src[j] >> (8 * e)) & 31u);
                                ++at;
                            }
                        }
                    }
                }
                uint32_t thr = tE;
                CFGMS_K2_MARK(5);  // list built
                if (any_overflow) {
#pragma unroll
                    for (int j = 0; j < CPL; ++j) {
                        uint32_t ovf_mask = __ballot_sync(0xffffffffu, j * 32 + lane < G && (key[j][3] | 31u) >= tE);
                        while (ovf_mask && n_list >= 0) {
                            // up to four overflowing chunks per round: their 128-byte rows are requested together,
                            // so a cell with several of them pays one L2 round trip, not one per chunk
                            int cc[4];
                            float zv[4];
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                cc[u] = ovf_mask ? j * 32 + __ffs(ovf_mask) - 1 : -1;
                                ovf_mask &= ovf_mask - 1u;        // 0 stays 0
                                zv[u] = cc[u] >= 0 ? __ldcg(zr + cc[u] * 32 + lane) : 0.f;
                            }
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                if (cc[u] < 0 || n_list < 0) continue;
                                const uint32_t k32 = float_key(zv[u]);
                                const bool pred = k32 >= tE;
                                const uint32_t b = __ballot_sync(0xffffffffu, pred);
                                if (n_list + __popc(b) > cap) { n_list = -1; continue; }   // too many ties: full scan
                                if (pred) {
                                    const int pos = n_list + __popc(b & ((1u << lane) - 1u));
                                    list_key[pos] = k32;
                                    list_v[pos] = tok0 + cc[u] * 32 + lane;
                                }
                                n_list += __popc(b);
                            }
                        }
                    }
                    __syncwarp();
                    if (n_list > tk) {
                        // More than k values >= t_E: a re-read chunk revealed values its four emitted ones had
                        // hidden (or several values tie at t_E).  The completed set holds every z >= t_E, so the
                        // exact threshold is its k-th largest: drop the (n_list - k) smallest.  (Deciding this by
                        // the list length, not by per-chunk bookkeeping, stays exact when a chunk's 4th emitted
                        // value shares t_E's 27-bit bucket but lies below t_E.)
                        const int extra = n_list - tk;
                        if (extra <= 8) {
                            for (int it = 0;; ++it) {
                                uint32_t mine_min = 0xffffffffu;
                                int mine_pos = 0;
                                for (int e = lane; e < n_list; e += 32) {
                                    const uint32_t ck = list_key[e];
                                    if (list_v[e] >= 0 && ck < mine_min) { mine_min = ck; mine_pos = e; }
                                }
                                thr = __reduce_min_sync(0xffffffffu, mine_min);
                                if (it == extra) break;
                                const uint32_t holder = __ballot_sync(0xffffffffu, mine_min == thr);
                                if (lane == __ffs(holder) - 1) list_v[mine_pos] = -1 - list_v[mine_pos];   // drop one instance
                                __syncwarp();
                            }
                            // dropped entries are <= thr; those tying it still survive (threshold semantics)
                            for (int e = lane; e < n_list; e += 32)
                                if (list_v[e] < 0) list_v[e] = -1 - list_v[e];
                            __syncwarp();
                        } else {
                            thr = warp_radix_select(SmemKeys{list_key}, n_list, tk, hist, lane);
                        }
                    }
                }
                __syncwarp();
                CFGMS_K2_MARK(6);  // overflow chunks handled, exact threshold known
                if (n_list >= 0) {
                    // two list entries per lane and iteration, so that their Philox / logarithm chains overlap
                    for (int e = lane; e < n_list; e += 64) {
                        const int e2 = e + 32 < n_list ? e + 32 : e;
                        const uint32_t ka = list_key[e], kb = list_key[e2];
                        const int va = list_v[e], vb = list_v[e2];
                        const bool sa = ka >= thr, sb = e2 != e && kb >= thr;
                        if (greedy) {
                            if (sa) best_update(best, key_float(ka), va);
                            if (sb) best_update(best, key_float(kb), vb);
                        } else if (sa || sb) {
                            const float ga = gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, va);
                            const float gb = gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, vb);
                            if (sa) best_update(best, key_float(ka) + ga, va);
                            if (sb) best_update(best, key_float(kb) + gb, vb);
                        }
                    }
                } else {
                    const uint32_t thr_full = warp_radix_select(GlobalKeys{zr}, V, tk, hist, lane);
                    for (int v = lane; v < V; v += 32) {
                        const float zv = __ldcg(zr + v);
                        if (float_key(zv) >= thr_full)
                            best_update(best, greedy ? zv + 0.0f : zv + 0.0f + gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, tok0 + v), tok0 + v);
                    }
                }
            }
        } else {
            // no top-k filter, or k larger than the emitted set: scan the whole row from the spill
            uint32_t thr_full = 0u;
            if (filter) thr_full = warp_radix_select(GlobalKeys{zr}, V, tk, hist, lane);
            for (int v = lane; v < V; v += 32) {
                const float zv = __ldcg(zr + v);
                if (float_key(zv) >= thr_full)
                    best_update(best, zv + 0.0f + gumbel_noise(p.seed_lo, p.seed_hi, req, tau, gi, tok0 + v), tok0 + v);
            }
        }
        best = warp_argmax(best);
        token = best.v;
        CFGMS_K2_MARK(7);          // noise drawn, argmax done
    }
    if (valid && lane == 0) write_cell(p, r, i, pm, cp, token, modality);
    xchg_finish(p);
    CFGMS_K2_MARK(8);
    CFGMS_K2_MARK(15);
    if (p.ready) {
        // the last CTA to finish re-arms the counters for the next step's K1 (which starts after this grid)
        __syncthreads();
        if (threadIdx.x == 0 && atomicAdd(p.done, 1) == static_cast<int>(gridDim.x) - 1) {
            for (int g = 0; g < p.S * p.num_row_blocks; ++g) p.ready[g] = 0;
            *p.done = 0;
        }
    }
}

}  // namespace cfgms
