// K1 — head projection + CFG merge + temperature + per-chunk candidate pass (rows a1-a2 and
// the first part of a3 of DESIGN.md's hot-path table; Eq. 1).
//
// Orientation ("swap-AB", B200-first): the head weights are the M operand and the batch rows
// are the N operand of tcgen05.mma, so one accumulator tile is
//     D[v][r] = sum_k W[n0 + v][k] * H[r0 + r][k],   v in [0,128) TMEM lanes, r in [0,BN) columns.
// Consequences:
//   * every weight byte is fetched from HBM once when R <= 256 (one CTA owns a 128-token slice
//     of the concatenated vocabulary S*V for ALL rows) — the decode regime is weight streaming;
//   * the cond row and its uncond companion are ADJACENT TMEM COLUMNS, i.e. adjacent registers
//     of the same thread after tcgen05.ld: Eq. 1 is two FMAs per merged logit, no shuffles;
//   * per-token bias (W_i e_i, folded at create) is one scalar per thread;
//   * an epilogue warp owns 32 consecutive tokens (its TMEM lane quarter) = exactly one
//     candidate chunk, so the chunk's selection needs no cross-warp traffic;
//   * the z spill is written with 32 consecutive tokens per warp store (128 B coalesced).
//
// kPair: two CTAs of a cluster (same TPC) run ONE tcgen05.mma.cta_group::2 of M = 256: each CTA
// brings its own 128-token weight tile and HALF of the batch-row tile, which halves the
// shared-memory fill and read traffic of the row operand (the limiter of the one-CTA kernel at
// large batches).  Each CTA's epilogue reads its own 128 accumulator lanes from its own TMEM.
//
// Warp roles (352 threads, persistent over tiles, 1 CTA/SM):
//   warp 0, 2   TMA producers: warp 0 the W tile [128 x 64], warp 2 the H tile [BN (or BN/2) x 64] bf16 -> 128B-swizzled ring
//   warp 1      TMEM allocator + single-thread tcgen05.mma issuer (leader CTA only when kPair),
//               2 accumulator stages in TMEM so the epilogue of tile t overlaps the mainloop of t+1
//   warps 3-10  epilogue, two warps per TMEM lane quarter (alternate 64-column slab pairs):
//               tcgen05.ld -> merge -> x 1/temp -> z spill (fp32) -> per-chunk top-4 candidates
//
// Register budget: the register file is split over the SM's four sub-partitions (16 K registers
// each) and the eleven warps land 3/3/3/2 on them.  At 168 registers per thread a three-warp
// sub-partition is full (16128 of 16384), so NO warp of any other grid can become resident on the
// SM (measured: even a 32-thread kernel waits for this one to exit; setmaxnreg.dec does not help,
// it returns registers to the CTA's own pool only).  Capped at 152, every sub-partition keeps
// >= 1792 registers free = one 48..56-register warp of the finalize kernel (K2), which is what
// lets K2's CTAs sit beside this kernel and sample finished (stream, row block) groups while
// the GEMM is still running.
#pragma once
#include "ptx_sm100.cuh"
#include "finalize.cuh"   // gumbel_noise (the epilogue-noise measurement probe of the -DCFGMS_PROBES build)

namespace cfgms {

constexpr int kBM = 128;        // vocabulary rows per CTA tile (UMMA M, or half of M = 256 when paired)
constexpr int kBK = 64;         // K elements per stage (128 B = swizzle span)
constexpr int kMaxBN = 256;     // batch rows per tile (UMMA N)
constexpr int kEpiWarps = 8;
constexpr int kCtrlWarps = 3;     // TMA producer (weights), MMA issuer, TMA producer (hidden rows)
constexpr int kGemmMaxRegs = 152; // see "Register budget" above
constexpr int kGemmThreads = 32 * (kCtrlWarps + kEpiWarps);
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;
constexpr int kCoefSlots = 512; // two-row slots whose coefficients fit the shared-memory table (R <= 1024)
constexpr int kStgPitch = 33;   // words; +1 keeps both access patterns of the transpose conflict-free

// Per two-row slot: out0 = c00*acc[2j] + c01*acc[2j+1] + bias*d0 (request at the even row);
// out1 = c11*acc[2j+1] + bias*d1 (only when the slot holds two unpaired rows).
struct __align__(16) SlotCoefA {
    float c00, c01, d0;
    int kind;                 // bit0: even row owns a request; bit1: odd row owns its own request
};
struct __align__(16) SlotCoefB {
    float c11, d1;
    float m00, m01;           // pre-temperature merge weights for the debug tap
};

struct GemmParams {
    int R, NT, d, BN, num_row_blocks, num_vocab_tiles, num_tiles, num_kb, stages;
    int row0;            // batch row of this launch's first row: the host-buffer entry point launches the GEMM once per
                         // uploaded row block (rows [row0, row0 + R) of the batch; the hidden-state tensor map covers
                         // exactly those rows), everything else launches it once with row0 = 0
    const int32_t* pair_map;
    const float* w;
    const float* temp;
    const int32_t* phase; // nullable [R]: request phase (include/cfgms.h); the CFG merge runs in the audio phase only
    const float* bias;   // [NT]
    float* z;            // [R][NT]
    float* tap;          // nullable [R][NT]
    float* cand_val;     // nullable [R][NT/32][4]: four z of every 32-token chunk, descending (see below)
    uint32_t* cand_src;  // nullable [R][NT/32]: their token offsets inside the chunk, 8 bits each
    int* err;            // sticky error word {code | row << 8}
    int* ready;          // nullable [S][num_row_blocks]: epilogue-warp arrivals per (stream, row block), see K2
    int V;               // tokens per stream (ready != nullptr requires V % kBM == 0)
    int split_tma;       // 1: warp 2 issues the row-tile loads; 0: warp 0 issues both (warp 2 idles)
    int split_k;         // 1, or 2: one-wave GEMMs run on four-CTA clusters, two CTA pairs each taking half of K (kSplit build)
#ifdef CFGMS_PROBES
    // Measurement probes for the two design choices DESIGN.md section 7 argues.  They exist only in the probe build of
    // the library (-DCFGMS_PROBES, libcfgms_probes.so, `bench.py --probes`); the product build has neither the fields
    // nor the code:
    //   probe bit 0: draw the Philox-Gumbel noise of EVERY merged logit in this epilogue (north_star's literal
    //                fusion) — the draws are folded into a sink word, results are unchanged: a lower bound of what
    //                the fused variant costs;
    //   probe bit 1: do not write the z spill (timing only: cells that need a spilled row sample garbage).
    int probe;
    uint32_t* probe_sink;
#endif
    uint64_t policy_w, policy_h;
#ifdef CFGMS_TRACE
    unsigned long long* trace;
#endif
};

struct GemmSmemLayout {
    // dynamic smem (1024-aligned): A ring | B ring | coefA | coefB | barriers | candidate transpose
    __host__ __device__ static constexpr uint32_t a_bytes() { return kBM * kBK * 2; }
    __host__ __device__ static constexpr uint32_t b_bytes(int rows) { return static_cast<uint32_t>(rows) * kBK * 2; }
    __host__ __device__ static constexpr uint32_t coef_bytes() { return kCoefSlots * (sizeof(SlotCoefA) + sizeof(SlotCoefB)); }
    // transpose stage: 16 requests x 32 tokens per epilogue warp; the split-K build also receives its partner's 4 KB of
    // partial sums there, so it keeps 32 rows
    __host__ __device__ static constexpr uint32_t stg_bytes(bool split) { return kEpiWarps * (split ? 32 : 16) * kStgPitch * 4; }
    __host__ __device__ static constexpr uint32_t misc_bytes(bool split) { return coef_bytes() + 256 + stg_bytes(split); }
    __host__ __device__ static constexpr uint32_t total(int b_rows, int stages, bool split) {
        return 1024 + stages * (a_bytes() + b_bytes(b_rows)) + misc_bytes(split);
    }
};

// Slot coefficients from pair_map / w / temp (DESIGN.md batch layout contract).
__device__ __forceinline__ void make_slot_coef(const GemmParams& p, int r0, SlotCoefA& a, SlotCoefB& b) {
    a = {0.f, 0.f, 0.f, 0};
    b = {0.f, 0.f, 0.f, 0.f};
    const int r1 = r0 + 1;          // r0, r1: rows of the BATCH (pair_map holds batch rows)
    const int r_end = p.row0 + p.R;
    if (r0 >= r_end) return;
    const int pm0 = p.pair_map[r0];
    const int pm1 = r1 < r_end ? p.pair_map[r1] : -1;
    const float t0 = p.temp[r0];
    const float it0 = t0 == 0.f ? 1.f : 1.f / t0;
    if (pm0 == r1 && pm1 == r0) {                       // (cond, uncond) pair: Eq. 1
        // "this CFG merge operates only during the audio phase; it bypasses modality-switching
        // tokens": outside the audio phase the request's logits are its conditional row's (w = 1 in Eq. 1)
        const float w = (p.phase && __ldcg(p.phase + r0) != 2 /* CFGMS_PHASE_AUDIO */) ? 1.f : p.w[r0];
        a.c00 = w * it0; a.c01 = (1.f - w) * it0; a.d0 = it0; a.kind = 1;
        b.m00 = w; b.m01 = 1.f - w;
    } else if (pm0 == -1 && pm1 == -1) {                // two unpaired rows
        a.c00 = it0; a.d0 = it0; a.kind = 1;
        b.m00 = 1.f;
        if (r1 < r_end) {
            const float t1 = p.temp[r1];
            const float it1 = t1 == 0.f ? 1.f : 1.f / t1;
            b.c11 = it1; b.d1 = it1;
            a.kind = 3;
        }
    } else {                                            // contract violated
        atomicCAS(p.err, 0, 3 /* CFGMS_ERR_LAYOUT */ | (r0 << 8));
    }
}

// Per-chunk candidate pass (north_star step 3, "per-N-tile top-k candidate pass held in warp
// registers").  The warp's 32 tokens x 32 requests block is transposed through a warp-private
// shared-memory stage; afterwards two lanes share a request's chunk of 32 z values.  They keep
// the four largest as PACKED keys (order-preserving 27-bit float key | 5-bit reversed token
// offset) with 7 integer min/max per value — no predicates, no index bookkeeping — then
// re-reads the four exact values and emits them sorted (descending, lowest token first).
// Selection granularity is the 27-bit key bucket: a value that is NOT emitted has
//     float_key(hidden) <= float_key(smallest emitted) | 31,
// which is the bound K2 uses to decide whether a chunk may hide a top-k member.
// TWO lanes per request (a warp finishes 16 requests x 32 tokens per slab): lane
// `part` (0 / 1) scans tokens [16 part, 16 part + 16) of the request's chunk, the two sorted packed-key lists are
// merged through one shuffle each (the four largest of two descending lists a, b are max(a[i], b[3 - i]); packed
// keys are distinct inside a chunk), and both lanes finish with the chunk's result.  Every lane of the warp calls it.
__device__ __forceinline__ void chunk_top4_two_lanes(const float* col, int part, float (&val)[4], uint32_t& src) {
    uint32_t t0 = 0u, t1 = 0u, t2 = 0u, t3 = 0u;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int idx = 16 * part + e;
        const uint32_t u = __float_as_uint(col[idx]);
        const uint32_t s = static_cast<uint32_t>(static_cast<int32_t>(u) >> 31);
        uint32_t pk = ((u ^ (s | 0x80000000u)) | 31u) ^ static_cast<uint32_t>(idx);
        uint32_t m;
        m = min(t0, pk); t0 = max(t0, pk); pk = m;
        m = min(t1, pk); t1 = max(t1, pk); pk = m;
        m = min(t2, pk); t2 = max(t2, pk); pk = m;
        t3 = max(t3, pk);
    }
    const uint32_t b0 = __shfl_xor_sync(0xffffffffu, t0, 16), b1 = __shfl_xor_sync(0xffffffffu, t1, 16);
    const uint32_t b2 = __shfl_xor_sync(0xffffffffu, t2, 16), b3 = __shfl_xor_sync(0xffffffffu, t3, 16);
    uint32_t c0 = max(t0, b3), c1 = max(t1, b2), c2 = max(t2, b1), c3 = max(t3, b0);
    int ix[4] = {static_cast<int>((c0 & 31u) ^ 31u), static_cast<int>((c1 & 31u) ^ 31u),
                 static_cast<int>((c2 & 31u) ^ 31u), static_cast<int>((c3 & 31u) ^ 31u)};
#pragma unroll
    for (int j = 0; j < 4; ++j) val[j] = col[ix[j]];
    // exact order: value descending, token ascending (the four are an unordered set here: full 4-sorter, then
    // one more exchange of the middle pair is already part of the 5-comparator network)
#define CFGMS_CX(a, b)                                                                   \
    {                                                                                    \
        const bool sw = (val[b] > val[a]) || (val[b] == val[a] && ix[b] < ix[a]);        \
        const float tv = sw ? val[b] : val[a]; val[b] = sw ? val[a] : val[b]; val[a] = tv; \
        const int ti = sw ? ix[b] : ix[a];    ix[b] = sw ? ix[a] : ix[b];    ix[a] = ti; \
    }
    CFGMS_CX(0, 1) CFGMS_CX(2, 3) CFGMS_CX(0, 2) CFGMS_CX(1, 3) CFGMS_CX(1, 2)
#undef CFGMS_CX
    src = static_cast<uint32_t>(ix[0]) | (static_cast<uint32_t>(ix[1]) << 8) | (static_cast<uint32_t>(ix[2]) << 16) |
          (static_cast<uint32_t>(ix[3]) << 24);
}

// One 32-column slab (16 two-row slots x 32 tokens: lane = token, v[2 j], v[2 j + 1] = the accumulators of slot j's two
// rows) from accumulators to outputs: CFG merge + bias + 1 / temperature, the z spill, and the candidate pass (transpose
// through `stg`, two lanes per request).  Pass A serves the request at the even row of every slot, pass B the request at
// the odd row of slots that hold two unpaired rows.  Branch-free inner loops: predicated stores, one running row
// pointer, coefficients preloaded by the caller — so the unrolled loops pipeline instead of serialising on a load, a
// branch and a store per slot.
template <bool kTap, bool kCand>
__device__ __forceinline__ void finish_slab(const GemmParams& p, const uint32_t (&v)[32], const SlotCoefA (&c)[16],
                                            const SlotCoefA* ca, const SlotCoefB* cb, float* stg, int row_base, int n, int nb,
                                            bool n_ok, bool chunk_ok, float bias, int lane, bool allow_a, bool allow_b) {
    const size_t NT = static_cast<size_t>(p.NT);
    char* zp = reinterpret_cast<char*>(p.z + static_cast<size_t>(row_base) * NT + n);
    float* tp = kTap ? p.tap + static_cast<size_t>(row_base) * NT + n : nullptr;
    const size_t row_stride = 2 * NT * sizeof(float);         // bytes between the even rows of two slots
#ifdef CFGMS_PROBES
    const bool spill = n_ok && !(p.probe & 2);
#else
    const bool spill = n_ok;
#endif
    const int o = lane & 15, part = lane >> 4;                // candidate pass: request o of the warp's 16, token half `part`
    int any_kind = 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) any_kind |= c[j].kind;
    const bool pass_a = allow_a && (any_kind & 1) != 0;
    const bool pass_b = allow_b && (any_kind & 2) != 0;
    if (pass_a) {
        char* zq = zp;
        asm volatile("" : "+l"(zq));
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const float a0 = __uint_as_float(v[2 * j]), a1 = __uint_as_float(v[2 * j + 1]);
            const float z0 = fmaf(c[j].c00, a0, fmaf(c[j].c01, a1, bias * c[j].d0));
            const bool own = (c[j].kind & 1) != 0;
            st_global_f32_if(zq, z0, own && spill);
            zq += row_stride;
            if (kTap && own && n_ok) { const SlotCoefB t = cb[j]; tp[static_cast<size_t>(2 * j) * NT] = fmaf(t.m00, a0, fmaf(t.m01, a1, bias)); }
            if (kCand) stg[j * kStgPitch + lane] = (own && n_ok) ? z0 + 0.0f : -INFINITY;
        }
#ifdef CFGMS_PROBES
        if (kCand && (p.probe & 1)) {
            // measurement probe: the noise of every merged logit of the slab, drawn here (rolled loop over the staged z
            // values so that the product path's code stays as it is); the draws are folded into a sink word
            uint32_t sink = 0u;
#pragma unroll 1
            for (int j = 0; j < 16; ++j)
                sink ^= __float_as_uint(stg[j * kStgPitch + lane] +
                                        gumbel_noise(0x1234u, 0x5678u, static_cast<uint32_t>(row_base + 2 * j), 7, n >> 11, n & 2047));
            if (sink == 0x9e3779b9u) *p.probe_sink = sink;    // keeps the draws alive
        }
#endif
        if (kCand) {
            __syncwarp();
            float val[4]; uint32_t src;
            chunk_top4_two_lanes(stg + o * kStgPitch, part, val, src);
            if ((ca[o].kind & 1) && chunk_ok && part == 0) {
                const size_t chunk = (static_cast<size_t>(row_base + 2 * o) * NT + nb) >> 5;
                *reinterpret_cast<float4*>(p.cand_val + chunk * 4) = make_float4(val[0], val[1], val[2], val[3]);
                p.cand_src[chunk] = src;
            }
            __syncwarp();
        }
    }
    if (pass_b) {
        char* zq = zp + NT * sizeof(float);
        asm volatile("" : "+l"(zq));
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const SlotCoefB t = cb[j];
            const float a1 = __uint_as_float(v[2 * j + 1]);
            const float z1 = fmaf(t.c11, a1, bias * t.d1);
            const bool own = (c[j].kind & 2) != 0;
            st_global_f32_if(zq, z1, own && spill);
            zq += row_stride;
            if (kTap && own && n_ok) tp[static_cast<size_t>(2 * j + 1) * NT] = a1 + bias;
            if (kCand) stg[j * kStgPitch + lane] = (own && n_ok) ? z1 + 0.0f : -INFINITY;
        }
        if (kCand) {
            __syncwarp();
            float val[4]; uint32_t src;
            chunk_top4_two_lanes(stg + o * kStgPitch, part, val, src);
            if ((ca[o].kind & 2) && chunk_ok && part == 0) {
                const size_t chunk = (static_cast<size_t>(row_base + 2 * o + 1) * NT + nb) >> 5;
                *reinterpret_cast<float4*>(p.cand_val + chunk * 4) = make_float4(val[0], val[1], val[2], val[3]);
                p.cand_src[chunk] = src;
            }
            __syncwarp();
        }
    }
}

template <bool kTap, bool kCand, bool kPair, bool kSplit = false, int EW = kEpiWarps>
__device__ __forceinline__ void head_gemm_body(const CUtensorMap& tmap_w, const CUtensorMap& tmap_h, const GemmParams& p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int stages = p.stages;
    const int BN = p.BN;
    const int b_rows = kPair ? BN / 2 : BN;          // batch rows this CTA stages per K block
    const uint32_t a_bytes = GemmSmemLayout::a_bytes();
    const uint32_t b_bytes = GemmSmemLayout::b_bytes(b_rows);
    const uint32_t smem_a = smem_base;
    const uint32_t smem_b = smem_a + stages * a_bytes;
    const uint32_t smem_coef_a = smem_b + stages * b_bytes;
    const uint32_t smem_coef_b = smem_coef_a + kCoefSlots * sizeof(SlotCoefA);
    const uint32_t bar_base = smem_coef_b + kCoefSlots * sizeof(SlotCoefB);
    // barriers: full[8] | empty[8] | tmem_full[2] | tmem_empty[2] | tmem base pointer | 8 B spare | xchg[8]   (8 B each)
    const uint32_t bar_full = bar_base;
    const uint32_t bar_empty = bar_base + 8 * kMaxStages;
    const uint32_t bar_tfull = bar_base + 16 * kMaxStages;
    const uint32_t bar_tempty = bar_tfull + 16;
    const uint32_t tmem_ptr_smem = bar_tempty + 16;
    const uint32_t bar_xchg = bar_tempty + 32;        // split-K: one per epilogue warp (partial sums received)
    const uint32_t smem_stg = bar_base + 256;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    SlotCoefA* coef_a = reinterpret_cast<SlotCoefA*>(smem_gen + (smem_coef_a - smem_base));
    SlotCoefB* coef_b = reinterpret_cast<SlotCoefB*>(smem_gen + (smem_coef_b - smem_base));
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem_gen + (tmem_ptr_smem - smem_base));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    // Cluster layout: one CTA; or a CTA pair (ranks 0, 1); or, split-K, two pairs (ranks 0, 1 | 2, 3) that work on the
    // same tile, pair `ks` taking K blocks [ks * kb_half, (ks + 1) * kb_half).
    static_assert(!kSplit || kPair, "split-K runs on CTA pairs");
    const uint32_t cluster_rank = kPair ? cluster_ctarank() : 0u;
    const uint32_t cta_rank = cluster_rank & 1u;              // rank inside the pair
    const uint32_t leader_rank = cluster_rank & ~1u;          // cluster rank of this pair's leader
    const uint16_t pair_mask = static_cast<uint16_t>(3u << leader_rank);
    const int ks = kSplit ? static_cast<int>(cluster_rank >> 1) : 0;
    const bool leader = cta_rank == 0u;
    const int cta_shift = kSplit ? 2 : kPair ? 1 : 0;
    const int worker = static_cast<int>(blockIdx.x >> cta_shift);
    const int num_workers = static_cast<int>(gridDim.x >> cta_shift);
    const int kb_half = kSplit ? (p.num_kb + 1) >> 1 : p.num_kb;
    const int kb_begin = ks * kb_half;
    const int kb_end = min(p.num_kb, kb_begin + kb_half);

    if (threadIdx.x == 0) { CFGMS_TRACE_MARK(p.trace, 0); CFGMS_TRACE_MARK(p.trace, 1); }
    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap_w);
        tma_prefetch_desc(&tmap_h);
        for (int s = 0; s < stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull + 8 * a, 1);
            mbar_init(bar_tempty + 8 * a, EW * (kPair ? 2 : 1));
        }
        if (kSplit)
            for (int w = 0; w < EW; ++w) mbar_init(bar_xchg + 8 * w, 1);
        fence_barrier_init();
    }
    if (warp == 1) {
        if (kPair) { tmem_alloc_pair(tmem_ptr_smem, kTmemCols); tmem_relinquish_pair(); }
        else { tmem_alloc(tmem_ptr_smem, kTmemCols); tmem_relinquish(); }
    }
    tc_fence_before();
    if (kPair) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    if (threadIdx.x == 0) CFGMS_TRACE_MARK(p.trace, 2);          // set-up done
    // This grid may itself have been launched early, as a programmatic dependent of whatever precedes it in
    // the stream (the previous step's finalize kernel, or the kernel that produced the hidden states): its
    // launch latency and the set-up above then overlap that kernel's tail.  Each warp role executes
    // griddepcontrol.wait (pdl_wait_primary) right before its first access to data another kernel may
    // produce or still read; the weight producer never needs to (the head weights are constant for the
    // context's lifetime, include/cfgms.h), so weight tiles start streaming before the previous kernel ends.

    if (warp == 2 && !p.split_tma) {
        // idle: warp 0 issues both loads (see below); wait at the teardown barrier
    } else if (warp == 0 || warp == 2) {
        // ================= TMA producers (every CTA): warp 0 loads the weight tiles, warp 2 the row tiles ====
        // Two issuing warps where the GEMM is short (one or two waves: configs 2-4 gain 3-5 %); a long,
        // power-capped GEMM (config 5) measured ~3 % slower with the extra spinning warp, so there warp 0
        // issues both loads and warp 2 idles (p.split_tma).
        // The whole warp walks the loop (warp-uniform state stays in uniform registers); one
        // elected lane issues.  Transaction bytes of both CTAs land on the leader's barrier; the
        // weight producer of the leader posts the expected byte count of the whole stage.
        const bool load_w = warp == 0;
        const bool load_h = warp == 2 || !p.split_tma;
        if (load_h) pdl_wait_primary();        // the hidden states may come from the preceding kernel
        if (load_h && lane == 0) CFGMS_TRACE_MARK(p.trace, 3);   // previous kernel done (row producer)
        const uint32_t full_sig = kPair ? mapa_shared(bar_full, leader_rank) : bar_full;
        const uint32_t tx_bytes = (a_bytes + b_bytes) * (kPair ? 2u : 1u);
        int s = 0;
        uint32_t phase = 0;
        for (int tile = worker; tile < p.num_tiles; tile += num_workers) {
            const int rb = tile % p.num_row_blocks;
            const int vp = tile / p.num_row_blocks;
            const int vt = kPair ? vp * 2 + static_cast<int>(cta_rank) : vp;
            const int row0 = rb * BN + static_cast<int>(cta_rank) * b_rows;
            for (int kb = kb_begin; kb < kb_end; ++kb) {
                mbar_wait(bar_empty + 8 * s, phase ^ 1, p.err, 1);
                if (elect_one()) {
                    if (load_w) {
                        if (leader) mbar_arrive_expect_tx(bar_full + 8 * s, tx_bytes);
                        if (kPair) tma_load_2d_pair(smem_a + s * a_bytes, &tmap_w, full_sig + 8 * s, kb * kBK, vt * kBM, p.policy_w);
                        else tma_load_2d(smem_a + s * a_bytes, &tmap_w, full_sig + 8 * s, kb * kBK, vt * kBM, p.policy_w);
                    }
                    if (load_h) {
                        if (kPair) tma_load_2d_pair(smem_b + s * b_bytes, &tmap_h, full_sig + 8 * s, kb * kBK, row0, p.policy_h);
                        else tma_load_2d(smem_b + s * b_bytes, &tmap_h, full_sig + 8 * s, kb * kBK, row0, p.policy_h);
                    }
                }
                __syncwarp();
                if (++s == stages) { s = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (leader CTA) =================
        // This loop paces the tensor pipe: 4 MMAs of 128 cycles per K block, so it must stay far
        // below 512 cycles per iteration — whole-warp control flow, one elected lane issues.
        if (leader) {
            const uint32_t idesc = umma_idesc_bf16_f32(kPair ? 2 * kBM : kBM, BN);
            const uint64_t a_desc0 = umma_smem_desc_sw128(smem_a);
            const uint64_t b_desc0 = umma_smem_desc_sw128(smem_b);
            int s = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int tile = worker; tile < p.num_tiles; tile += num_workers) {
                mbar_wait(bar_tempty + 8 * acc, acc_phase ^ 1, p.err, 2);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * BN;
                for (int kb = kb_begin; kb < kb_end; ++kb) {
                    mbar_wait(bar_full + 8 * s, phase, p.err, 3);
                    tc_fence_after();
                    if (lane == 0 && tile == worker && kb == kb_begin) CFGMS_TRACE_MARK(p.trace, 4);                  // first stage landed
                    if (lane == 0 && tile == worker && kb == (kb_begin + kb_end) / 2) CFGMS_TRACE_MARK(p.trace, 5);   // half of the first tile
                    if (lane == 0 && tile == worker && kb == kb_end - 1) CFGMS_TRACE_MARK(p.trace, 6);                // last stage of the first tile landed
                    if (elect_one()) {
                        // the start-address field counts 16-byte units
                        const uint64_t a_desc = a_desc0 + static_cast<uint64_t>((s * a_bytes) >> 4);
                        const uint64_t b_desc = b_desc0 + static_cast<uint64_t>((s * b_bytes) >> 4);
#pragma unroll
                        for (int k = 0; k < kBK / 16; ++k) {
                            // advance 16 bf16 = 32 B along K inside the swizzle span: +2 in the >>4 field
                            const uint32_t accum = (kb != kb_begin || k != 0) ? 1u : 0u;
                            if (kPair) umma_bf16_pair(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                            else umma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                        }
                        if (kPair) umma_commit_pair(bar_empty + 8 * s, pair_mask); else umma_commit(bar_empty + 8 * s);
                        if (kb == kb_end - 1) {
                            if (kPair) umma_commit_pair(bar_tfull + 8 * acc, pair_mask); else umma_commit(bar_tfull + 8 * acc);
                        }
                    }
                    __syncwarp();
                    if (++s == stages) { s = 0; phase ^= 1; }
                }
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
            }
        }
    } else if (kSplit) {
        // ================= split-K epilogue (warps 3..10, every CTA): one tile per cluster ============================
        // The pair of K half `ks` OWNS batch columns [64 ks, 64 ks + 64) of the 128-column tile.  Epilogue warp
        // (quarter, half) hands the 32 columns [64 (1 - ks) + 32 half, + 32) of its TMEM lane quarter to the same warp
        // of the CTA that holds the same vocabulary rows in the other pair (cluster rank ^ 2) and finishes its own 32
        // columns, so the eight warps of all four CTAs share the epilogue evenly.  The partial sums travel as
        // asynchronous DSMEM stores into the receiving warp's (still unused) transpose stage and complete on that
        // warp's own mbarrier: no cluster-wide barrier, no fence, and nothing touches a TMA ring that may still be busy.
        const int ew = warp - kCtrlWarps;
        const int quarter = warp & 3;
        const int half = ew >> 2;
        const int et = ew * 32 + lane;
        const uint32_t xbar = bar_xchg + 8 * ew;
        if (lane == 0) mbar_arrive_expect_tx(xbar, 4096);
        pdl_wait_primary();
        pdl_launch_dependents();
        for (int slot = et; slot < p.num_row_blocks * (BN / 2); slot += 32 * EW) {   // the host guarantees it fits
            SlotCoefA ca; SlotCoefB cb;
            make_slot_coef(p, p.row0 + 2 * slot, ca, cb);
            coef_a[slot] = ca; coef_b[slot] = cb;
        }
        const int tile = worker;
        const int rb = tile % p.num_row_blocks;
        const int vt = (tile / p.num_row_blocks) * 2 + static_cast<int>(cta_rank);
        // Batches of at most 64 rows fill only columns [0, 64): there the pair of K half `ks` owns the 32 columns
        // [32 ks, 32 ks + 32) and its two warps per lane quarter split the two passes over them (half 0: the requests
        // at even rows, half 1: those at odd rows of unpaired slots), so that a CFG-off batch does not leave one pair
        // idle while the other runs both passes.
        const bool narrow = p.R <= 64;
        const int col0 = narrow ? 32 * ks : 64 * ks + 32 * half;                 // first owned column of this warp
        const int send_col = narrow ? 32 * (1 - ks) : 64 * (1 - ks) + 32 * half; // first column handed to the other pair
        const int nb = vt * kBM + quarter * 32;               // first token of this warp's chunk
        const int n = nb + lane;
        const bool n_ok = n < p.NT;
        const bool chunk_ok = nb < p.NT;
        const float bias = n_ok ? __ldg(p.bias + n) : 0.f;
        named_bar_sync(1, 32 * EW);
        mbar_wait(bar_tfull, 0, p.err, 4);
        tc_fence_after();
        if (warp == kCtrlWarps && lane == 0) CFGMS_TRACE_MARK(p.trace, 7);
        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
        const uint32_t stg_addr = smem_stg + static_cast<uint32_t>(ew) * (32 * kStgPitch * 4);
        float* stg = reinterpret_cast<float*>(smem_gen + (stg_addr - smem_base));
        uint32_t v[32];
        {
            uint32_t xs[32];
            tmem_ld_32x32b_x32(taddr + send_col, xs);
            tmem_ld_wait();
            tmem_ld_32x32b_x32(taddr + col0, v);
            const uint32_t dst = mapa_shared(stg_addr + static_cast<uint32_t>(lane) * 16u, cluster_rank ^ 2u);   // [col / 4][lane][4]
            const uint32_t dbar = mapa_shared(xbar, cluster_rank ^ 2u);
#pragma unroll
            for (int j = 0; j < 8; ++j)
                st_async_cluster_v4(dst + 512u * j, xs[4 * j], xs[4 * j + 1], xs[4 * j + 2], xs[4 * j + 3], dbar);
            tmem_ld_wait();
        }
        if (warp == kCtrlWarps && lane == 0) CFGMS_TRACE_MARK(p.trace, 12);     // partial sums sent
        const int row_base = p.row0 + rb * BN + col0;
        const SlotCoefA* ca = coef_a + rb * (BN / 2) + (col0 >> 1);
        const SlotCoefB* cb = coef_b + rb * (BN / 2) + (col0 >> 1);
        SlotCoefA c[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) c[j] = ca[j];
        mbar_wait_cluster(xbar, 0, p.err, 5);
        if (warp == kCtrlWarps && lane == 0) CFGMS_TRACE_MARK(p.trace, 13);     // partner's partial sums landed
        {
            const float4* rx = reinterpret_cast<const float4*>(stg) + lane;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float4 r = rx[32 * j];
                v[4 * j] = __float_as_uint(__uint_as_float(v[4 * j]) + r.x);
                v[4 * j + 1] = __float_as_uint(__uint_as_float(v[4 * j + 1]) + r.y);
                v[4 * j + 2] = __float_as_uint(__uint_as_float(v[4 * j + 2]) + r.z);
                v[4 * j + 3] = __float_as_uint(__uint_as_float(v[4 * j + 3]) + r.w);
            }
        }
        __syncwarp();                                             // the stage is reused for the transpose below
        finish_slab<kTap, kCand>(p, v, c, ca, cb, stg, row_base, n, nb, n_ok, chunk_ok, bias, lane, !narrow || half == 0,
                                 !narrow || half == 1);
        if (warp == kCtrlWarps && lane == 0) { CFGMS_TRACE_MARK(p.trace, 8); CFGMS_TRACE_MARK(p.trace, 9); }
    } else {
        // ================= epilogue, slab form (warps 3 .. 3 + EW - 1, every CTA) =================
        // EW / 4 warps per TMEM lane quarter walk the tile's 32-column slabs; every slab goes through finish_slab (the
        // branch-free form written for the split-K epilogue): 13 k instead of 20 k cycles per 192-row tile of config 4.
        // (Twelve or sixteen epilogue warps at 128 / 96 registers measured no faster / slower than eight at 146.)
        pdl_wait_primary();
        pdl_launch_dependents();
        const int ew = warp - kCtrlWarps;
        const int quarter = warp & 3;
        const int sub = ew >> 2;                  // which of the quarter's EW / 4 warps
        constexpr int WPQ = EW / 4;
        const int et = ew * 32 + lane;
        float* stg = reinterpret_cast<float*>(smem_gen + (smem_stg - smem_base)) + ew * (16 * kStgPitch);
        const int n_slab = BN / 32;
        const int slots_per_rb = BN / 2;
        const uint32_t tempty_sig = (kPair && !leader) ? mapa_shared(bar_tempty, leader_rank) : bar_tempty;
        const bool full_table = p.num_row_blocks * slots_per_rb <= kCoefSlots;
        if (full_table) {
            // coefficients of every slot, once (the first mainloop hides it)
            for (int slot = et; slot < p.num_row_blocks * slots_per_rb; slot += 32 * EW) {
                SlotCoefA ca; SlotCoefB cb;
                make_slot_coef(p, p.row0 + 2 * slot, ca, cb);
                coef_a[slot] = ca; coef_b[slot] = cb;
            }
            named_bar_sync(1, 32 * EW);
        }
        int acc = 0;
        uint32_t acc_phase = 0;
        int cur_rb = -1;
        for (int tile = worker; tile < p.num_tiles; tile += num_workers) {
            const int rb = tile % p.num_row_blocks;
            const int vp = tile / p.num_row_blocks;
            const int vt = kPair ? vp * 2 + static_cast<int>(cta_rank) : vp;
            if (!full_table && rb != cur_rb) {            // more than 1024 rows: the table holds one row block at a time
                named_bar_sync(1, 32 * EW);               // everyone finished reading the old table
                if (et < slots_per_rb) {
                    SlotCoefA ca; SlotCoefB cb;
                    make_slot_coef(p, p.row0 + rb * BN + 2 * et, ca, cb);
                    coef_a[et] = ca; coef_b[et] = cb;
                }
                named_bar_sync(1, 32 * EW);
                cur_rb = rb;
            }
            const int slot_base = full_table ? rb * slots_per_rb : 0;
            const int nb = vt * kBM + quarter * 32;       // first token of this warp's chunk
            const int n = nb + lane;
            const bool n_ok = n < p.NT;
            const bool chunk_ok = nb < p.NT;
            const float bias = n_ok ? __ldg(p.bias + n) : 0.f;
            mbar_wait(bar_tfull + 8 * acc, acc_phase, p.err, 4);
            tc_fence_after();
            if (warp == kCtrlWarps && lane == 0 && tile == worker) CFGMS_TRACE_MARK(p.trace, 7);      // first accumulator complete
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + acc * BN;
            if (sub >= n_slab) {                          // nothing to read for this warp: release at once
                tc_fence_before();
                __syncwarp();
                if (lane == 0) { if (kPair && !leader) mbar_arrive_cluster(tempty_sig + 8 * acc); else mbar_arrive(bar_tempty + 8 * acc); }
            }
            for (int sl = sub; sl < n_slab; sl += WPQ) {
                uint32_t v[32];
                tmem_ld_32x32b_x32(taddr + sl * 32, v);
                const SlotCoefA* ca = coef_a + slot_base + sl * 16;
                const SlotCoefB* cb = coef_b + slot_base + sl * 16;
                SlotCoefA c[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) c[j] = ca[j];
                tmem_ld_wait();
                if (sl + WPQ >= n_slab) {                 // this warp's share of the accumulator stage is in registers
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) { if (kPair && !leader) mbar_arrive_cluster(tempty_sig + 8 * acc); else mbar_arrive(bar_tempty + 8 * acc); }
                }
                finish_slab<kTap, kCand>(p, v, c, ca, cb, stg, p.row0 + rb * BN + sl * 32, n, nb, n_ok, chunk_ok, bias, lane, true, true);
            }
            if (p.ready && vt * kBM < p.NT) {
                __syncwarp();
                if (lane == 0) red_release_gpu_add(p.ready + ((vt * kBM) / p.V) * p.num_row_blocks + rb, 1);
            }
            if (warp == kCtrlWarps && lane == 0 && tile == worker) CFGMS_TRACE_MARK(p.trace, 8);      // first epilogue done
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
        if (warp == kCtrlWarps && lane == 0) CFGMS_TRACE_MARK(p.trace, 9);
    }

    tc_fence_before();
    // (split-K: nothing is published through this barrier — it keeps the four CTAs alive until every one of them has
    // received its partner's partial sums and is done with the pair's tensor memory — so it carries no release fence,
    // which would wait for the logit stores above to drain)
    if (kSplit) cluster_sync_relaxed(); else if (kPair) cluster_sync_all(); else __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        if (kPair) tmem_dealloc_pair(tmem_base, kTmemCols); else tmem_dealloc(tmem_base, kTmemCols);
    }
    if (threadIdx.x == 0) { CFGMS_TRACE_MARK(p.trace, 10); CFGMS_TRACE_MARK(p.trace, 15); }
}

// Full register budget (168): the fastest GEMM, but nothing else fits on its SMs while it runs.
template <bool kTap, bool kCand, bool kPair>
__global__ void __launch_bounds__(kGemmThreads, 1)
cfgms_head_gemm_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_h,
                       const GemmParams p) {
    head_gemm_body<kTap, kCand, kPair>(tmap_w, tmap_h, p);
}

// Split-K build for one-wave GEMMs (clusters of four CTAs; the host chooses it, see choose_row_tile in cfgms.cu).
template <bool kTap, bool kCand>
__global__ void __launch_bounds__(kGemmThreads, 1)
cfgms_head_gemm_splitk_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_h,
                              const GemmParams p) {
    head_gemm_body<kTap, kCand, true, true>(tmap_w, tmap_h, p);
}

// Lean register budget (see "Register budget" above): leaves room for the finalize kernel's CTAs on
// the same SMs; used when K2 is launched as a programmatic dependent of a multi-wave GEMM.
template <bool kTap, bool kPair>
__global__ void __maxnreg__(kGemmMaxRegs)
cfgms_head_gemm_lean_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_h,
                            const GemmParams p) {
    head_gemm_body<kTap, true, kPair>(tmap_w, tmap_h, p);
}

}  // namespace cfgms
