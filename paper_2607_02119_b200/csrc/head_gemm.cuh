// K1 — head projection + CFG merge + temperature (rows a1-a2 and the first part of a3 of
// DESIGN.md's hot-path table; Eq. 1).
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
//   * the z spill is written with 32 consecutive tokens per warp store (128 B coalesced).
//
// Warp roles (192 threads, persistent over tiles, 1 CTA/SM):
//   warp 0      TMA producer: W tile [128 x 64] + H tile [BN x 64] bf16 -> 128B-swizzled smem ring
//   warp 1      TMEM allocator + single-thread tcgen05.mma issuer (M=128, N=BN, K=16), 2 accumulator
//               stages in TMEM so the epilogue of tile t overlaps the mainloop of tile t+1
//   warps 2-5   epilogue: tcgen05.ld -> merge -> x 1/temp -> z[row][n] (fp32) (+ debug tap)
#pragma once
#include "ptx_sm100.cuh"

namespace cfgms {

constexpr int kBM = 128;        // vocabulary rows per tile (UMMA M)
constexpr int kBK = 64;         // K elements per stage (128 B = swizzle span)
constexpr int kMaxBN = 256;     // batch rows per tile (UMMA N)
constexpr int kGemmThreads = 192;
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;

// Per two-row slot coefficients: out0 = c00*acc[2j] + c01*acc[2j+1] + bias*d0 (request at the
// even row), out1 = c11*acc[2j+1] + bias*d1 (only when the slot holds two unpaired rows).
struct __align__(16) SlotCoef {
    float c00, c01, d0, c11;
    float d1, m00, m01;       // m00/m01: pre-temperature merge weights for the debug tap
    int kind;                 // bit0: even row owns a request; bit1: odd row owns its own request
};

struct GemmParams {
    int R, NT, d, BN, num_row_blocks, num_vocab_tiles, num_tiles, num_kb, stages;
    const int32_t* pair_map;
    const float* w;
    const float* temp;
    const float* bias;   // [NT]
    float* z;            // [R][NT]
    float* tap;          // nullable [R][NT]
    float* cand_val;     // nullable [R][NT/32][4]: top-4 z of every 32-token chunk, descending
    uint32_t* cand_src;  // nullable [R][NT/32]: their lane offsets inside the chunk, 8 bits each
    int* err;            // sticky error word {code | row << 8}
    uint64_t policy_w, policy_h;
};

struct GemmSmemLayout {
    // dynamic smem (1024-aligned): A ring | B ring | coefficients | barriers | tmem ptr
    __host__ __device__ static constexpr uint32_t a_bytes() { return kBM * kBK * 2; }
    __host__ __device__ static constexpr uint32_t b_bytes(int BN) { return static_cast<uint32_t>(BN) * kBK * 2; }
    __host__ __device__ static constexpr uint32_t coef_bytes() { return (kMaxBN / 2) * sizeof(SlotCoef); }
    __host__ __device__ static constexpr uint32_t stage_bytes() { return 32 * (kBM + 1) * 4; }  // candidate transpose
    __host__ __device__ static constexpr uint32_t misc_bytes() { return coef_bytes() + 256 + stage_bytes(); }
    __host__ __device__ static constexpr uint32_t total(int BN, int stages) {
        return 1024 + stages * (a_bytes() + b_bytes(BN)) + misc_bytes();
    }
};

// Per-chunk candidate pass (north_star step 3, "per-N-tile top-k candidate pass held in
// registers").  In this orientation a thread owns ONE token and many requests, the wrong axis
// for a per-request top-k, so every 32-column accumulator slab is transposed through a 16 KB
// shared-memory stage: afterwards epilogue thread (o, q) owns output column o (one request)
// and the 32 tokens of vocabulary chunk q of the tile, and keeps the chunk's four largest z
// (descending, lowest token first among equals) in registers with plain compares/selects.
constexpr int kStageCols = 32;                 // output columns staged per round
constexpr int kStagePitch = kBM + 1;           // words; +1 keeps both access patterns conflict-free
__device__ __forceinline__ void top4_insert(float x, int e, float (&t)[4], int (&ix)[4]) {
    const bool c0 = x > t[0], c1 = x > t[1], c2 = x > t[2], c3 = x > t[3];
    t[3] = c2 ? t[2] : (c3 ? x : t[3]);   ix[3] = c2 ? ix[2] : (c3 ? e : ix[3]);
    t[2] = c1 ? t[1] : (c2 ? x : t[2]);   ix[2] = c1 ? ix[1] : (c2 ? e : ix[2]);
    t[1] = c0 ? t[0] : (c1 ? x : t[1]);   ix[1] = c0 ? ix[0] : (c1 ? e : ix[1]);
    t[0] = c0 ? x : t[0];                 ix[0] = c0 ? e : ix[0];
}

template <bool kTap, bool kCand>
__global__ void __launch_bounds__(kGemmThreads, 1)
cfgms_head_gemm_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_h,
                       const GemmParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int stages = p.stages;
    const uint32_t a_bytes = GemmSmemLayout::a_bytes();
    const uint32_t b_bytes = GemmSmemLayout::b_bytes(p.BN);
    const uint32_t smem_a = smem_base;
    const uint32_t smem_b = smem_a + stages * a_bytes;
    const uint32_t smem_coef = smem_b + stages * b_bytes;
    const uint32_t bar_base = smem_coef + GemmSmemLayout::coef_bytes();
    // barriers: full[stages], empty[stages], tmem_full[2], tmem_empty[2]  (8 B each)
    const uint32_t bar_full = bar_base;
    const uint32_t bar_empty = bar_base + 8 * kMaxStages;
    const uint32_t bar_tfull = bar_base + 16 * kMaxStages;
    const uint32_t bar_tempty = bar_tfull + 16;
    const uint32_t tmem_ptr_smem = bar_tempty + 16;
    const uint32_t smem_stage = bar_base + 256;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    SlotCoef* coef = reinterpret_cast<SlotCoef*>(smem_gen + (smem_coef - smem_base));
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem_gen + (tmem_ptr_smem - smem_base));
    float* stage = reinterpret_cast<float*>(smem_gen + (smem_stage - smem_base));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap_w);
        tma_prefetch_desc(&tmap_h);
        for (int s = 0; s < stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull + 8 * a, 1);
            mbar_init(bar_tempty + 8 * a, 4);
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        tmem_alloc(tmem_ptr_smem, kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    const int BN = p.BN;
    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            int s = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
                const int rb = tile % p.num_row_blocks;
                const int vt = tile / p.num_row_blocks;
                for (int kb = 0; kb < p.num_kb; ++kb) {
                    mbar_wait(bar_empty + 8 * s, phase ^ 1, p.err, 1);
                    mbar_arrive_expect_tx(bar_full + 8 * s, a_bytes + b_bytes);
                    tma_load_2d(smem_a + s * a_bytes, &tmap_w, bar_full + 8 * s, kb * kBK, vt * kBM, p.policy_w);
                    tma_load_2d(smem_b + s * b_bytes, &tmap_h, bar_full + 8 * s, kb * kBK, rb * BN, p.policy_h);
                    if (++s == stages) { s = 0; phase ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ================= MMA issuer =================
        if (lane == 0) {
            const uint32_t idesc = umma_idesc_bf16_f32(kBM, BN);
            int s = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
                mbar_wait(bar_tempty + 8 * acc, acc_phase ^ 1, p.err, 2);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * BN;
                for (int kb = 0; kb < p.num_kb; ++kb) {
                    mbar_wait(bar_full + 8 * s, phase, p.err, 3);
                    tc_fence_after();
                    const uint64_t a_desc = umma_smem_desc_sw128(smem_a + s * a_bytes);
                    const uint64_t b_desc = umma_smem_desc_sw128(smem_b + s * b_bytes);
#pragma unroll
                    for (int k = 0; k < kBK / 16; ++k) {
                        // advance 16 bf16 = 32 B along K inside the swizzle span: +2 in the >>4 field
                        umma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
                    }
                    umma_commit(bar_empty + 8 * s);
                    if (++s == stages) { s = 0; phase ^= 1; }
                }
                umma_commit(bar_tfull + 8 * acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
            }
        }
        __syncwarp();
    } else {
        // ================= epilogue (warps 2..5) =================
        const int quarter = warp & 3;             // TMEM lane quarter this warp may read
        const int et = (warp - 2) * 32 + lane;    // 0..127 index among epilogue threads
        int acc = 0;
        uint32_t acc_phase = 0;
        int cur_rb = -1;
        for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
            const int rb = tile % p.num_row_blocks;
            const int vt = tile / p.num_row_blocks;
            if (rb != cur_rb) {
                // slot coefficients of this row block: one slot per epilogue thread
                named_bar_sync(1, 128);           // everyone finished reading the old table
                const int slot = et;
                if (slot < BN / 2) {
                    const int r0 = rb * BN + 2 * slot, r1 = r0 + 1;
                    SlotCoef c = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0};
                    if (r0 < p.R) {
                        const int pm0 = p.pair_map[r0];
                        const int pm1 = r1 < p.R ? p.pair_map[r1] : -1;
                        const float t0 = p.temp[r0];
                        const float it0 = t0 == 0.f ? 1.f : 1.f / t0;
                        if (pm0 == r1 && pm1 == r0) {                       // (cond, uncond) pair: Eq. 1
                            const float w = p.w[r0];
                            c.c00 = w * it0; c.c01 = (1.f - w) * it0; c.d0 = it0;
                            c.m00 = w; c.m01 = 1.f - w;
                            c.kind = 1;
                        } else if (pm0 == -1 && pm1 == -1) {                // two unpaired rows
                            c.c00 = it0; c.d0 = it0; c.m00 = 1.f;
                            c.kind = 1;
                            if (r1 < p.R) {
                                const float t1 = p.temp[r1];
                                const float it1 = t1 == 0.f ? 1.f : 1.f / t1;
                                c.c11 = it1; c.d1 = it1;
                                c.kind = 3;
                            }
                        } else {                                            // contract violated
                            atomicCAS(p.err, 0, 3 /* CFGMS_ERR_LAYOUT */ | (r0 << 8));
                        }
                    }
                    coef[slot] = c;
                }
                named_bar_sync(1, 128);
                cur_rb = rb;
            }
            const int n = vt * kBM + quarter * 32 + lane;
            const bool n_ok = n < p.NT;
            const float bias = n_ok ? __ldg(p.bias + n) : 0.f;

            mbar_wait(bar_tfull + 8 * acc, acc_phase, p.err, 4);
            tc_fence_after();
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + acc * BN;
            const int nchunks = BN / 32;
            for (int c = 0; c < nchunks; ++c) {
                uint32_t v[32];
                tmem_ld_32x32b_x32(taddr + c * 32, v);
                tmem_ld_wait();
                if (c == nchunks - 1) {
                    // accumulator stage fully read into registers: hand it back to the MMA warp
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_tempty + 8 * acc);
                }
                const int row_base = rb * BN + c * 32;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const SlotCoef sc = coef[c * 16 + j];
                    const float a0 = __uint_as_float(v[2 * j]);
                    const float a1 = __uint_as_float(v[2 * j + 1]);
                    const int r0 = row_base + 2 * j;
                    const int kind = sc.kind;
                    if (n_ok && (kind & 1)) {
                        const float z0 = fmaf(sc.c00, a0, fmaf(sc.c01, a1, bias * sc.d0));
                        p.z[static_cast<size_t>(r0) * p.NT + n] = z0;
                        if (kTap) p.tap[static_cast<size_t>(r0) * p.NT + n] = fmaf(sc.m00, a0, fmaf(sc.m01, a1, bias));
                        if (kCand) stage[(2 * j) * kStagePitch + quarter * 32 + lane] = z0 + 0.0f;
                    }
                    if (n_ok && (kind & 2)) {
                        const float z1 = fmaf(sc.c11, a1, bias * sc.d1);
                        p.z[static_cast<size_t>(r0 + 1) * p.NT + n] = z1;
                        if (kTap) p.tap[static_cast<size_t>(r0 + 1) * p.NT + n] = a1 + bias;
                        if (kCand) stage[(2 * j + 1) * kStagePitch + quarter * 32 + lane] = z1 + 0.0f;
                    }
                }
                if (kCand) {
                    named_bar_sync(2, 128);                 // slab staged by all four epilogue warps
                    const int o = et & 31;                  // output column of the slab
                    const int q = et >> 5;                  // vocabulary chunk of the tile
                    const int kind_o = coef[c * 16 + (o >> 1)].kind;
                    const int nb = vt * kBM + q * 32;       // first token of the chunk (NT % 32 == 0)
                    if (((kind_o >> (o & 1)) & 1) && nb < p.NT) {
                        float t[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
                        int ix[4] = {0, 0, 0, 0};
                        const float* col = stage + o * kStagePitch + q * 32;
#pragma unroll
                        for (int e = 0; e < 32; ++e) top4_insert(col[e], e, t, ix);
                        const size_t chunk = (static_cast<size_t>(row_base + o) * p.NT + nb) >> 5;
                        *reinterpret_cast<float4*>(p.cand_val + chunk * 4) = make_float4(t[0], t[1], t[2], t[3]);
                        p.cand_src[chunk] = static_cast<uint32_t>(ix[0]) | (static_cast<uint32_t>(ix[1]) << 8) |
                                            (static_cast<uint32_t>(ix[2]) << 16) | (static_cast<uint32_t>(ix[3]) << 24);
                    }
                    named_bar_sync(2, 128);                 // stage may be overwritten
                }
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, kTmemCols);
    }
}

}  // namespace cfgms
