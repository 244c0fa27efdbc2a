// Host side of libcfgms.so: the C ABI declared in include/cfgms.h.  Validation, TMA tensor-map
// encoding, tile-shape choice, launches.  No torch types, no CPU fallback.
#include "../../include/cfgms.h"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "aux_kernels.cuh"
#include "finalize.cuh"
#include "head_gemm.cuh"

using namespace cfgms;

// Measurement probes are not part of the C ABI: the two flag bits exist only in the probe build
// (`python -m paper_2607_02119_b200.build --probes` -> libcfgms_probes.so, used by `bench.py --probes`).  The product
// build refuses them, so that a probe run against the wrong library fails instead of timing the product path.
#define CFGMS_CFG_PROBE_EPILOGUE_NOISE 256u /* the head GEMM's epilogue also draws the Philox-Gumbel noise of EVERY merged logit */
#define CFGMS_CFG_PROBE_NO_SPILL 512u       /* the head GEMM does not write the fp32 logit spill (timing only: wrong tokens)    */

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr int kProfMax = 4096;
constexpr int kOverlapMinWaves = 3;

struct HostStage {  // device staging for the *_host entry points
    void* hidden = nullptr;
    char* params = nullptr;        // device: one block for every small per-row input of a step (one H2D copy)
    char* params_pinned = nullptr; // pinned host mirror the caller's arrays are packed into
    size_t params_bytes = 0;
    int32_t *tokens = nullptr, *frame = nullptr, *frame_index = nullptr;
    cudaStream_t copy_stream = nullptr;   // hidden-state row blocks are uploaded here while the GEMM of the previous block runs
    cudaEvent_t chunk_ev[16] = {nullptr};
    int32_t* deint_in = nullptr;
    int32_t* deint_out = nullptr;
    size_t deint_in_bytes = 0, deint_out_bytes = 0;
};

}  // namespace

struct cfgms_ctx {
    int S = 0, d = 0, V = 0, NT = 0;
    int device = 0, num_sms = 0;
    int max_rows = 0, pad_token = 0, row_tile_override = 0, max_stages = 0;
    int stream_base = 0, stream_stride = 1;   // stream-sharded heads: global stream of local stream i
    int S_total = 0;                  // streams of the whole head (== S unless stream-sharded); 0 = unknown (sharded, not given)
    int V_text = 0, n_bridge = 0;     // phase state machine (cfgms_set_phase_table)
    int32_t bridge[16] = {0};
    int poll_ns = 2000;       // K2's sleep between polls of a ready counter: 1-4 us measured ~2.4 % faster than 50-200 ns at config 5
    int pair_mode = 0;                // 0 = chosen per step, 1 = never pair CTAs, 2 = always pair
    int split_mode = 0;               // split-K for one-wave GEMMs: 0 = chosen per step, 1 = never
    int max_clusters4 = 0;            // four-CTA clusters of the split-K kernel that can be co-resident on this device
    bool pdl_finalize = true;         // serial mode: launch a small K2 grid as a programmatic dependent of K1
#ifdef CFGMS_PROBES
    int probe = 0;                    // measurement probes (CFGMS_CFG_PROBE_*), see GemmParams::probe
#endif
    const __nv_bfloat16* heads = nullptr;
    float* bias = nullptr;            // [NT] what the epilogue adds: bias_base (+ the caller's logit bias)
    float* bias_base = nullptr;       // [NT] W_i e_i, folded at create
    float* z = nullptr;               // [max_rows][NT]
    float* cand_val = nullptr;        // [max_rows][NT/32][4] top-4 per 32-token chunk (candidate path)
    uint32_t* cand_src = nullptr;     // [max_rows][NT/32]
    bool use_cand = false;            // V % 32 == 0 && V <= 8192
    __nv_bfloat16* hidden_bf16 = nullptr;  // [max_rows][d], used when the caller passes fp32
    int* err = nullptr;               // device: sticky {code | row << 8}
    int* ready = nullptr;             // device: [S][row blocks] K1 -> K2 tile arrivals, then one `done` counter
    int ready_words = 0;
    bool overlap = false;             // K2 may run as a programmatic dependent of K1 (candidate path, V % 128 == 0)
    int overlap_mode = 0;             // 0 = when the GEMM has >= kOverlapMinWaves waves, 1 = never, 2 = whenever eligible
    EncodeTiledFn encode = nullptr;
    CUtensorMap tmap_w;
    CUtensorMap tmap_h;
    const void* tmap_h_ptr = nullptr;
    int tmap_h_R = 0, tmap_h_box = 0;
    int max_smem_optin = 0;
    HostStage hs;
    bool hs_ready = false;
    // stream-sharded token exchange (cfgms_exchange_*): one device block [tokens | flags | state], symmetric on all ranks
    struct {
        int world = 0, rank = 0;
        void* base = nullptr;                 // this rank's block (cudaMalloc: exportable through CUDA IPC)
        size_t half_bytes = 0, latest_off = 0, flags_off = 0, state_off = 0;  // byte offsets inside every rank's block
        void* opened[64] = {nullptr};         // peers' blocks opened through IPC (closed at destroy)
        int32_t** d_tokens = nullptr;         // device arrays [world] of peer pointers
        uint32_t** d_flags = nullptr;
        bool connected = false;
    } xc;
    bool prof_on = false;
    cudaEvent_t* prof_ev = nullptr;   // [kProfMax][3]
    int prof_n = 0;
    cfgms_info info;
#ifdef CFGMS_TRACE
    unsigned long long* trace_k1 = nullptr;
    unsigned long long* trace_k2 = nullptr;
#endif
};

namespace {

int make_tmap_2d(cfgms_ctx* c, CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    // bf16 [rows][cols], cols contiguous; box = [box_rows][64] -> 128-byte swizzled smem rows
    cuuint64_t gdim[2] = {cols, rows};
    cuuint64_t gstride[1] = {cols * 2};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(kBK), box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = c->encode(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? CFGMS_OK : CFGMS_ERR_CUDA;
}

// Batch rows per accumulator tile (BN, a multiple of 64 = one slab pair of the epilogue, <= 256 =
// UMMA N with two accumulator stages in 512 TMEM columns) and whether two CTAs pair up on one
// M = 256 MMA.  A (cond, uncond) pair never straddles a tile because BN is even.
void choose_row_tile(const cfgms_ctx* c, int R, int* BN, int* nrb, bool* pair, bool* split) {
    const int vt = (c->NT + kBM - 1) / kBM;
    *split = false;
    // One-wave GEMMs (small batch x small vocabulary: the weight-streaming regime): when the (vocabulary
    // tile pair, 128-row block) tiles fill at most half of the CTA pairs, every tile is given to a cluster of FOUR CTAs,
    // two pairs that each stream half of K and exchange partial sums over DSMEM (head_gemm.cuh).  Against splitting
    // the rows instead (two 64-row blocks, each re-reading the weight tile from L2) this halves the bytes an SM
    // takes in (L2 -> SM is the wall there) and spreads the epilogue over all eight warps.
    if (c->split_mode != 1 && c->overlap_mode != 2 && c->row_tile_override == 0 && c->pair_mode != 1 && vt >= 2 && c->d >= 8 * kBK) {
        const int rb = (R + 127) / 128;
        const int tiles = ((vt + 1) / 2) * rb;
        if (rb * 64 <= kCoefSlots && tiles * 4 <= c->num_sms && tiles <= c->max_clusters4) {
            *BN = 128; *nrb = rb; *pair = true; *split = true;
            return;
        }
    }
    if (c->row_tile_override > 0) {
        *BN = c->row_tile_override;
        *nrb = (R + *BN - 1) / *BN;
    } else {
        // Cost model: a CTA's time for one tile is ~ the bytes it pulls per K step, (128 + BN) rows of
        // 128 B, and the slowest CTA runs ceil(tiles / SMs) tiles.  Splitting the rows re-reads the
        // weight tile from L2 (not HBM) but lets small batches occupy every SM.
        const int min_blocks = (R + kMaxBN - 1) / kMaxBN;
        long best_cost = -1;
        for (int blocks = min_blocks; blocks <= min_blocks * 8; ++blocks) {
            int per = (R + blocks - 1) / blocks;
            per = ((per + 63) / 64) * 64;
            const int nb = (R + per - 1) / per;
            const long waves = (static_cast<long>(vt) * nb + c->num_sms - 1) / c->num_sms;
            const long cost = waves * (kBM + per + 16);
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; *BN = per; *nrb = nb; }
            if (per <= 64) break;
        }
    }
    // Pairing halves the row-operand bytes every SM has to take in per K step (each CTA of the pair
    // stages half of the row tile).  It pays most in the tensor-bound regime (large row tiles), and
    // still measures 1-2 % faster at a 64-row tile (config 2: 19.85 vs 20.20 us/step), with the same CTA count.
    *pair = c->pair_mode == 2 || (c->pair_mode == 0 && *BN >= 64 && vt >= 2);
}

template <typename T>
int dev_alloc(T** p, size_t n) {
    return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T)) == cudaSuccess ? CFGMS_OK : CFGMS_ERR_NOMEM;
}

int validate_step(const cfgms_ctx* c, const cfgms_step_args* a) {
    if (!c || !a) return CFGMS_ERR_ARG;
    if (!a->hidden || !a->pair_map || !a->w || !a->temp || !a->top_k || !a->step || !a->tokens_out) return CFGMS_ERR_ARG;
    if (a->hidden_dtype != CFGMS_BF16 && a->hidden_dtype != CFGMS_F32) return CFGMS_ERR_ARG;
    if (a->R < 1) return CFGMS_ERR_ARG;
    if (a->R > c->max_rows) return CFGMS_ERR_SHAPE;
    if (a->delayed && a->T_cap < 1) return CFGMS_ERR_ARG;
    if ((a->frame_out || a->frame_index_out) && (!a->delayed || a->T_cap < c->S)) return CFGMS_ERR_ARG;
    if ((a->frame_out || a->frame_index_out) && (c->stream_base != 0 || c->stream_stride != 1)) return CFGMS_ERR_ARG;   // a frame needs every stream
    // the drain of a request ends S_global - 1 steps after its last frame: a shard must know S_global
    const bool state_out = a->step_next_out || a->n_frames_next_out || a->done_out || a->phase_next_out || a->phase_pos_next_out ||
                           a->modality_out;
    if ((a->step_next_out || a->n_frames_next_out || a->done_out || a->phase_next_out || a->phase_pos_next_out) && c->S_total == 0)
        return CFGMS_ERR_ARG;
    // The request state advances on what the PRIMARY stream (global stream 0) emitted, by the thread of that cell
    // (finalize.cuh write_cell).  A shard that does not hold global stream 0 has no such cell: refuse, rather than leave the
    // outputs silently unwritten and let a device-resident state loop on that rank run on stale state.
    if (state_out && c->stream_base != 0) return CFGMS_ERR_ARG;
    if (a->phase && (!a->phase_pos || a->force_token)) return CFGMS_ERR_ARG;
    if (!a->phase && (a->phase_pos || a->phase_next_out || a->phase_pos_next_out || a->modality_out)) return CFGMS_ERR_ARG;
    return CFGMS_OK;
}

}  // namespace

extern "C" {

const char* cfgms_strerror(int s) {
    switch (s) {
        case CFGMS_OK: return "ok";
        case CFGMS_ERR_ARG: return "invalid argument";
        case CFGMS_ERR_SHAPE: return "unsupported shape";
        case CFGMS_ERR_LAYOUT: return "pair_map violates the paired-slot layout contract";
        case CFGMS_ERR_CUDA: return "CUDA call failed";
        case CFGMS_ERR_ARCH: return "device is not sm_100 (no fallback path exists)";
        case CFGMS_ERR_NOMEM: return "out of device memory";
        case CFGMS_ERR_TIMEOUT: return "device-side pipeline wait timed out";
        case CFGMS_ERR_LIMIT: return "request exceeds the fixed scratch (CFGMS_STATIC_SCRATCH_BYTES) of a non-allocating entry point";
        default: return "unknown status";
    }
}

#ifdef CFGMS_PROBES
const char* cfgms_version(void) { return "cfgms 0.1 sm_100a (tcgen05/TMEM/TMA) +probes (measurement build, not the product), built " __DATE__; }
#else
const char* cfgms_version(void) { return "cfgms 0.1 sm_100a (tcgen05/TMEM/TMA), built " __DATE__; }
#endif

int cfgms_create(cfgms_ctx** out, const void* heads, const void* embeds, int32_t S, int32_t d, int32_t V,
                 const cfgms_config* cfg) {
    if (!out) return CFGMS_ERR_ARG;
    *out = nullptr;
    if (!heads || !embeds || S < 1 || d < 1 || V < 1) return CFGMS_ERR_ARG;
    if (S > 64 || (d % 8) != 0) return CFGMS_ERR_SHAPE;
    if (static_cast<int64_t>(S) * V > (1ll << 30)) return CFGMS_ERR_SHAPE;
    if ((reinterpret_cast<uintptr_t>(heads) & 15u) != 0) return CFGMS_ERR_ARG;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return CFGMS_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return CFGMS_ERR_CUDA;
    if (prop.major != 10) return CFGMS_ERR_ARCH;

    cfgms_ctx* c = new (std::nothrow) cfgms_ctx();
    if (!c) return CFGMS_ERR_NOMEM;
    c->S = S; c->d = d; c->V = V; c->NT = S * V;
    c->device = dev;
    c->num_sms = prop.multiProcessorCount;
    c->max_smem_optin = static_cast<int>(prop.sharedMemPerBlockOptin);
    c->max_rows = (cfg && cfg->max_rows > 0) ? cfg->max_rows : 1024;
    c->pad_token = (cfg && (cfg->flags & CFGMS_CFG_PAD_TOKEN)) ? cfg->pad_token : V;
    c->row_tile_override = cfg ? cfg->row_tile : 0;
    c->max_stages = (cfg && cfg->max_stages >= 2) ? cfg->max_stages : kMaxStages;
    if (cfg && cfg->stream_stride > 0) { c->stream_base = cfg->stream_base; c->stream_stride = cfg->stream_stride; }
    if (c->stream_base < 0) { delete c; return CFGMS_ERR_ARG; }
    const bool sharded = c->stream_base != 0 || c->stream_stride != 1;
    c->S_total = (cfg && cfg->global_streams > 0) ? cfg->global_streams : (sharded ? 0 : S);
    if (c->S_total != 0 && c->S_total < c->stream_base + (S - 1) * c->stream_stride + 1) { delete c; return CFGMS_ERR_ARG; }
    c->pair_mode = (cfg && (cfg->flags & CFGMS_CFG_SINGLE_CTA)) ? 1 : (cfg && (cfg->flags & CFGMS_CFG_CTA_PAIR)) ? 2 : 0;
    if (c->row_tile_override < 0 || c->row_tile_override > kMaxBN || (c->row_tile_override % 64) != 0) {
        delete c;
        return CFGMS_ERR_ARG;
    }
    c->heads = static_cast<const __nv_bfloat16*>(heads);
    c->use_cand = (V % 32 == 0) && V <= 8192 && !(cfg && (cfg->flags & CFGMS_CFG_NO_CANDIDATES));
    std::memset(&c->info, 0, sizeof(c->info));

    // the sampler keeps one row of V keys in shared memory
    if (static_cast<size_t>(V) * 4 + 4096 > static_cast<size_t>(c->max_smem_optin)) { delete c; return CFGMS_ERR_SHAPE; }

    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
        delete c;
        return CFGMS_ERR_CUDA;
    }
    c->encode = reinterpret_cast<EncodeTiledFn>(fn);

    int rc = CFGMS_OK;
    if ((rc = dev_alloc(&c->bias, static_cast<size_t>(c->NT))) != CFGMS_OK ||
        (rc = dev_alloc(&c->bias_base, static_cast<size_t>(c->NT))) != CFGMS_OK ||
        (rc = dev_alloc(&c->z, static_cast<size_t>(c->max_rows) * c->NT)) != CFGMS_OK ||
        (rc = dev_alloc(&c->hidden_bf16, static_cast<size_t>(c->max_rows) * d)) != CFGMS_OK ||
        (rc = dev_alloc(&c->err, 2)) != CFGMS_OK ||
        (c->use_cand && ((rc = dev_alloc(&c->cand_val, static_cast<size_t>(c->max_rows) * (c->NT / 32) * 4)) != CFGMS_OK ||
                         (rc = dev_alloc(&c->cand_src, static_cast<size_t>(c->max_rows) * (c->NT / 32))) != CFGMS_OK))) {
        cfgms_destroy(c);
        return rc;
    }
    cudaMemset(c->err, 0, 2 * sizeof(int));
    c->overlap_mode = (cfg && (cfg->flags & CFGMS_CFG_NO_OVERLAP)) ? 1 : (cfg && (cfg->flags & CFGMS_CFG_OVERLAP)) ? 2 : 0;
    c->pdl_finalize = !(cfg && (cfg->flags & CFGMS_CFG_NO_PDL_FINALIZE));
    c->split_mode = (cfg && (cfg->flags & CFGMS_CFG_NO_SPLIT_K)) ? 1 : 0;
#ifdef CFGMS_PROBES
    c->probe = (cfg && (cfg->flags & CFGMS_CFG_PROBE_EPILOGUE_NOISE) ? 1 : 0) | (cfg && (cfg->flags & CFGMS_CFG_PROBE_NO_SPILL) ? 2 : 0);
#else
    if (cfg && (cfg->flags & (CFGMS_CFG_PROBE_EPILOGUE_NOISE | CFGMS_CFG_PROBE_NO_SPILL))) { cfgms_destroy(c); return CFGMS_ERR_ARG; }
#endif
    c->overlap = c->use_cand && (V % kBM) == 0 && c->overlap_mode != 1;
    if (c->overlap) {
        c->ready_words = ((S * ((c->max_rows + 63) / 64) + 1 + 1) & ~1) + 32;   // counters | done | pad | stats (16 x u64)
        if ((rc = dev_alloc(&c->ready, static_cast<size_t>(c->ready_words))) != CFGMS_OK) {
            cfgms_destroy(c);
            return rc;
        }
        cudaMemset(c->ready, 0, static_cast<size_t>(c->ready_words) * sizeof(int));
    }

    if ((rc = make_tmap_2d(c, &c->tmap_w, heads, static_cast<uint64_t>(c->NT), static_cast<uint64_t>(d), kBM)) != CFGMS_OK) {
        cfgms_destroy(c);
        return rc;
    }

    // K4: bias[i][v] = sum_k W_i[v][k] e_i[k]
    {
        const int warps_per_block = 8;
        const int blocks = (c->NT + warps_per_block - 1) / warps_per_block;
        cfgms_bias_init_kernel<<<blocks, warps_per_block * 32>>>(c->heads, static_cast<const __nv_bfloat16*>(embeds),
                                                                  c->bias_base, S, V, d);
        cudaMemcpyAsync(c->bias, c->bias_base, static_cast<size_t>(c->NT) * sizeof(float), cudaMemcpyDeviceToDevice, 0);
        if (cudaDeviceSynchronize() != cudaSuccess) {
            cfgms_destroy(c);
            return CFGMS_ERR_CUDA;
        }
    }
    bool attr_ok = static_cast<int>(GemmSmemLayout::total(kMaxBN, 2, true)) <= c->max_smem_optin;
    auto set_smem = [&](const void* fn) {
        attr_ok = attr_ok && cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem_optin) == cudaSuccess;
    };
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<false, false, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<true, false, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<false, true, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<true, true, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<false, false, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<true, false, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<false, true, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_kernel<true, true, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_splitk_kernel<false, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_splitk_kernel<true, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_splitk_kernel<false, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_splitk_kernel<true, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_lean_kernel<false, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_lean_kernel<true, false>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_lean_kernel<false, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_head_gemm_lean_kernel<true, true>));
    set_smem(reinterpret_cast<const void*>(cfgms_finalize_cand_kernel<1>));
    set_smem(reinterpret_cast<const void*>(cfgms_finalize_cand_kernel<2>));
    set_smem(reinterpret_cast<const void*>(cfgms_finalize_cand_kernel<4>));
    set_smem(reinterpret_cast<const void*>(cfgms_finalize_cand_kernel<8>));
    if (!attr_ok) {
        cfgms_destroy(c);
        return CFGMS_ERR_CUDA;
    }
    {   // how many four-CTA clusters of the split-K kernel fit at once (GPC shapes decide; 0 disables split-K)
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3(4 * static_cast<unsigned>(c->num_sms / 4));
        lc.blockDim = dim3(kGemmThreads);
        lc.dynamicSmemBytes = static_cast<size_t>(c->max_smem_optin);
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 4; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        lc.attrs = at; lc.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, cfgms_head_gemm_splitk_kernel<false, true>, &lc) != cudaSuccess) { n = 0; cudaGetLastError(); }
        c->max_clusters4 = n;
    }
    if (cudaFuncSetAttribute(cfgms_finalize_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024) != cudaSuccess ||
        (V > 256 * 32 && cudaFuncSetAttribute(cfgms_finalize_large_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              static_cast<int>(static_cast<size_t>(V) * 4)) != cudaSuccess)) {
        cfgms_destroy(c);
        return CFGMS_ERR_CUDA;
    }
    cudaFuncSetAttribute(cfgms_deinterleave_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);

    c->info.S = S; c->info.d = d; c->info.V = V; c->info.max_rows = c->max_rows;
    c->info.pad_token = c->pad_token; c->info.num_sms = c->num_sms;
    c->info.vocab_tiles = (c->NT + kBM - 1) / kBM;
    *out = c;
    return CFGMS_OK;
}

void cfgms_destroy(cfgms_ctx* c) {
    if (!c) return;
    cudaFree(c->bias);
    cudaFree(c->bias_base);
    cudaFree(c->z);
    cudaFree(c->cand_val);
    cudaFree(c->cand_src);
    cudaFree(c->hidden_bf16);
    cudaFree(c->err);
    cudaFree(c->ready);
    for (int q = 0; q < 64; ++q)
        if (c->xc.opened[q]) cudaIpcCloseMemHandle(c->xc.opened[q]);
    cudaFree(c->xc.base);
    cudaFree(c->xc.d_tokens);
    cudaFree(c->xc.d_flags);
    if (c->prof_ev) {
        for (int j = 0; j < 3 * kProfMax; ++j)
            if (c->prof_ev[j]) cudaEventDestroy(c->prof_ev[j]);
        delete[] c->prof_ev;
    }
    HostStage& h = c->hs;
    cudaFree(h.hidden); cudaFree(h.params); cudaFreeHost(h.params_pinned);
    cudaFree(h.tokens); cudaFree(h.frame); cudaFree(h.frame_index); cudaFree(h.deint_in); cudaFree(h.deint_out);
    for (int j = 0; j < 16; ++j)
        if (h.chunk_ev[j]) cudaEventDestroy(h.chunk_ev[j]);
    if (h.copy_stream) cudaStreamDestroy(h.copy_stream);
    delete c;
}

}  // extern "C"

namespace {

// Host-buffer mode of a step (cfgms_step_host): the hidden states are still in (pinned) host memory; they are
// uploaded in two chunks of GEMM row blocks on a second stream, the second chunk while the GEMM of the first runs.
struct HostUpload {
    const char* host_hidden;   // bf16 [R][d] on the host
    char* dev_hidden;          // staging on the device
    int64_t* h2d_bytes;
};

int step_impl(cfgms_ctx* c, const cfgms_step_args* a, cudaStream_t st, const HostUpload* up) {
    int rc = CFGMS_OK;
    int launches = 0;

    // K5: fp32 hidden -> bf16 (RNE)
    const __nv_bfloat16* hidden = up ? reinterpret_cast<const __nv_bfloat16*>(up->dev_hidden) : static_cast<const __nv_bfloat16*>(a->hidden);
    if (!up && a->hidden_dtype == CFGMS_F32) {
        const size_t n = static_cast<size_t>(a->R) * c->d;
        if ((reinterpret_cast<uintptr_t>(a->hidden) & 15u) != 0) return CFGMS_ERR_ARG;
        const int blocks = static_cast<int>(std::min<size_t>((n / 4 + 255) / 256 + 1, static_cast<size_t>(c->num_sms) * 8));
        cfgms_cast_f32_bf16_kernel<<<blocks, 256, 0, st>>>(static_cast<const float*>(a->hidden), c->hidden_bf16, n);
        hidden = c->hidden_bf16;
        ++launches;
    }
    if ((reinterpret_cast<uintptr_t>(hidden) & 15u) != 0) return CFGMS_ERR_ARG;

    int BN, nrb;
    bool pair, split;
    choose_row_tile(c, a->R, &BN, &nrb, &pair, &split);
    if (up) {            // host-buffer mode launches the GEMM per row block: the plain tiling
        const int keep = c->split_mode;
        c->split_mode = 1;
        choose_row_tile(c, a->R, &BN, &nrb, &pair, &split);
        c->split_mode = keep;
    }
    const int b_rows = pair ? BN / 2 : BN;     // batch rows one CTA stages per K block (TMA box height)
    if (!up && (c->tmap_h_ptr != hidden || c->tmap_h_R != a->R || c->tmap_h_box != b_rows)) {
        rc = make_tmap_2d(c, &c->tmap_h, hidden, static_cast<uint64_t>(a->R), static_cast<uint64_t>(c->d),
                          static_cast<uint32_t>(b_rows));
        if (rc != CFGMS_OK) return rc;
        c->tmap_h_ptr = hidden; c->tmap_h_R = a->R; c->tmap_h_box = b_rows;
    }

    GemmParams gp;
    gp.R = a->R; gp.NT = c->NT; gp.d = c->d; gp.BN = BN;
    gp.num_row_blocks = nrb;
    gp.num_vocab_tiles = (c->NT + kBM - 1) / kBM;
    gp.num_tiles = (pair ? (gp.num_vocab_tiles + 1) / 2 : gp.num_vocab_tiles) * nrb;   // tiles of one worker (CTA or CTA pair)
    gp.num_kb = (c->d + kBK - 1) / kBK;
    const uint32_t stage_bytes = GemmSmemLayout::a_bytes() + GemmSmemLayout::b_bytes(b_rows);
    int stages = static_cast<int>((static_cast<uint32_t>(c->max_smem_optin) - 1024 - GemmSmemLayout::misc_bytes(split)) / stage_bytes);
    stages = std::max(2, std::min(stages, std::min(kMaxStages, c->max_stages)));
    gp.stages = stages;
    gp.pair_map = a->pair_map; gp.w = a->w; gp.temp = a->temp; gp.phase = a->phase;
    gp.bias = c->bias; gp.z = c->z; gp.tap = a->logits_out; gp.err = c->err;
    gp.cand_val = c->cand_val; gp.cand_src = c->cand_src;
    const int workers = split ? gp.num_tiles : std::min(gp.num_tiles, pair ? c->num_sms / 2 : c->num_sms);
    const bool prof = c->prof_on && c->prof_n < kProfMax;
    // Overlap K2 with K1 only where finished groups appear long before the GEMM ends (several waves of
    // tiles): a one- or two-wave GEMM has nothing to hide behind, and the lean register budget and
    // the polling finalize warps then cost more than the early launch saves (measured).
    // (While the profiling events are recorded the SAME kernels run, but K2 is launched strictly after K1 so
    // that each has a duration of its own.)
    const bool overlap = !up && !split && c->overlap && (c->overlap_mode == 2 || gp.num_tiles >= kOverlapMinWaves * workers);
    gp.ready = overlap ? c->ready : nullptr;
    gp.V = c->V;
#ifdef CFGMS_PROBES
    gp.probe = c->probe; gp.probe_sink = reinterpret_cast<uint32_t*>(c->err + 1);
#endif
    gp.split_tma = gp.num_tiles < kOverlapMinWaves * workers ? 1 : 0;
    gp.split_k = split ? 2 : 1;
    // weights are streamed (read by one CTA when there is a single row block) — unless the whole head is small enough to
    // stay in L2 from one step to the next; hidden is re-read by every CTA
    gp.policy_w = (nrb == 1 && static_cast<size_t>(c->NT) * c->d * 2 > (96u << 20)) ? kEvictFirst : kEvictNormal;
    gp.policy_h = kEvictLast;
    const int grid = split ? 4 * workers : pair ? 2 * workers : workers;
#ifdef CFGMS_TRACE
    gp.trace = c->trace_k1;
#endif
    size_t smem = GemmSmemLayout::total(b_rows, stages, split);
    if (overlap) {
        // The finalize kernel's CTAs must become resident BESIDE this kernel: cap the ring so that one of them fits, and ask
        // for the whole remainder — a smaller request lets the driver pick a smaller shared-memory carve-out for the SM
        // (196 KiB instead of 228), which leaves the finalize CTA no room at all (cfgms_overlap_stats then reads 0).
        const size_t k2_need = static_cast<size_t>(kCandWarps) * cand_warp_words(c->V) * 4 + 2048;
        const size_t budget = static_cast<size_t>(c->max_smem_optin) - k2_need;
        while (stages > 2 && GemmSmemLayout::total(b_rows, stages, split) > budget) --stages;
        gp.stages = stages;
        smem = std::max<size_t>(GemmSmemLayout::total(b_rows, stages, split), budget);
    }
    gp.row0 = 0;
    if (prof) cudaEventRecord(c->prof_ev[3 * c->prof_n + 0], st);
    // One launch for the whole batch — or, in host-buffer mode, one launch per uploaded chunk of row blocks: chunk k + 1
    // crosses PCIe while the GEMM of chunk k runs.
    // Two chunks: every launch streams the whole head once more, so fewer, larger launches win as long as the first GEMM
    // can start before the upload ends (config 5, 8 MiB over PCIe: 361 us/step with two chunks, 390 with four, 423 with one).
    const int cb = (nrb + 1) / 2;       // row blocks per uploaded chunk
    const int n_launch = up ? (nrb + cb - 1) / cb : 1;
    if (n_launch > 15) return CFGMS_ERR_SHAPE;      // chunk events 0..14 (15 orders the copy stream behind the caller's)
    for (int k = 0; k < n_launch; ++k) {
        CUtensorMap tmap_chunk;
        const CUtensorMap* tmap_h = &c->tmap_h;
        if (up) {
            HostStage& hs = c->hs;
            const int row0 = k * cb * BN, rows = std::min(cb * BN, a->R - row0);
            const size_t off = static_cast<size_t>(row0) * c->d * 2, bytes = static_cast<size_t>(rows) * c->d * 2;
            if (cudaMemcpyAsync(up->dev_hidden + off, up->host_hidden + off, bytes, cudaMemcpyHostToDevice, hs.copy_stream) != cudaSuccess ||
                cudaEventRecord(hs.chunk_ev[k], hs.copy_stream) != cudaSuccess ||
                cudaStreamWaitEvent(st, hs.chunk_ev[k], 0) != cudaSuccess)
                return CFGMS_ERR_CUDA;
            *up->h2d_bytes += static_cast<int64_t>(bytes);
            rc = make_tmap_2d(c, &tmap_chunk, up->dev_hidden + off, static_cast<uint64_t>(rows), static_cast<uint64_t>(c->d),
                              static_cast<uint32_t>(b_rows));
            if (rc != CFGMS_OK) return rc;
            tmap_h = &tmap_chunk;
            gp.row0 = row0; gp.R = rows; gp.num_row_blocks = (rows + BN - 1) / BN;
            gp.num_tiles = (pair ? (gp.num_vocab_tiles + 1) / 2 : gp.num_vocab_tiles) * gp.num_row_blocks;
        }
        const int launch_workers = split ? gp.num_tiles : std::min(gp.num_tiles, pair ? c->num_sms / 2 : c->num_sms);
        const int launch_grid = split ? 4 * launch_workers : pair ? 2 * launch_workers : launch_workers;
        using KernelFn = void (*)(const CUtensorMap, const CUtensorMap, const GemmParams);
        static const KernelFn table[8] = {
            cfgms_head_gemm_kernel<false, false, false>, cfgms_head_gemm_kernel<true, false, false>,
            cfgms_head_gemm_kernel<false, true, false>,  cfgms_head_gemm_kernel<true, true, false>,
            cfgms_head_gemm_kernel<false, false, true>,  cfgms_head_gemm_kernel<true, false, true>,
            cfgms_head_gemm_kernel<false, true, true>,   cfgms_head_gemm_kernel<true, true, true>};
        static const KernelFn lean[4] = {cfgms_head_gemm_lean_kernel<false, false>, cfgms_head_gemm_lean_kernel<true, false>,
                                         cfgms_head_gemm_lean_kernel<false, true>, cfgms_head_gemm_lean_kernel<true, true>};
        static const KernelFn splitk[4] = {cfgms_head_gemm_splitk_kernel<false, false>, cfgms_head_gemm_splitk_kernel<true, false>,
                                           cfgms_head_gemm_splitk_kernel<false, true>, cfgms_head_gemm_splitk_kernel<true, true>};
        const KernelFn fn = split ? splitk[(a->logits_out ? 1 : 0) | (c->use_cand ? 2 : 0)]
                          : overlap ? lean[(a->logits_out ? 1 : 0) | (pair ? 2 : 0)]
                                    : table[(a->logits_out ? 1 : 0) | (c->use_cand ? 2 : 0) | (pair ? 4 : 0)];
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3(static_cast<unsigned>(launch_grid));
        lc.blockDim = dim3(kGemmThreads);
        lc.dynamicSmemBytes = smem;
        lc.stream = st;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = split ? 4 : pair ? 2 : 1;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        // the GEMM may be launched while the previous kernel of the stream still runs (it waits for it on the
        // device before touching shared data, head_gemm.cuh): hides its launch latency and set-up
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = attr;
        lc.numAttrs = (c->overlap_mode == 1 || prof) ? 1 : 2;
        if (cudaLaunchKernelEx(&lc, fn, c->tmap_w, *tmap_h, gp) != cudaSuccess) return CFGMS_ERR_CUDA;
        ++launches;
    }
    if (prof) cudaEventRecord(c->prof_ev[3 * c->prof_n + 1], st);

    FinalizeParams fp;
    fp.R = a->R; fp.S = c->S; fp.V = c->V; fp.NT = c->NT;
    fp.z = c->z; fp.pair_map = a->pair_map; fp.temp = a->temp; fp.top_k = a->top_k; fp.step = a->step;
    fp.req_id = a->req_id; fp.n_frames = a->n_frames;
    fp.seed_lo = static_cast<uint32_t>(a->seed & 0xffffffffull);
    fp.seed_hi = static_cast<uint32_t>(a->seed >> 32);
    fp.pad_token = c->pad_token;
    fp.tokens_out = a->tokens_out; fp.delayed = a->delayed; fp.T_cap = a->T_cap;
    fp.cand_val = c->cand_val; fp.cand_src = c->cand_src;
    fp.force_token = a->force_token; fp.frame_out = a->frame_out; fp.frame_index_out = a->frame_index_out;
    fp.eos_token = a->eos_token; fp.step_next_out = a->step_next_out; fp.n_frames_next_out = a->n_frames_next_out;
    fp.done_out = a->done_out;
    fp.ready = gp.ready;
    fp.done = overlap ? c->ready + (c->ready_words - 33) : nullptr;
    fp.stats = overlap ? reinterpret_cast<unsigned long long*>(c->ready + (c->ready_words - 32)) : nullptr;
    fp.err = c->err;
    fp.BN = BN; fp.num_row_blocks = nrb;
    fp.magic_per_stream = fast_div_magic(2 * ((a->R + 1) / 2));
    fp.magic_bn = fast_div_magic(BN);
    fp.stream_base = c->stream_base; fp.stream_stride = c->stream_stride;
    fp.S_total = c->S_total > 0 ? c->S_total : c->S;
    fp.phase = a->phase; fp.phase_pos = a->phase_pos;
    fp.phase_next_out = a->phase_next_out; fp.phase_pos_next_out = a->phase_pos_next_out; fp.modality_out = a->modality_out;
    fp.V_text = c->V_text; fp.n_bridge = c->n_bridge;
    fp.xchg_tokens = c->xc.connected ? c->xc.d_tokens : nullptr;
    fp.xchg_flags = c->xc.connected ? c->xc.d_flags : nullptr;
    fp.xchg_state = c->xc.base ? reinterpret_cast<unsigned int*>(static_cast<char*>(c->xc.base) + c->xc.state_off) : nullptr;
    fp.xchg_world = c->xc.world; fp.xchg_rank = c->xc.rank;
    fp.xchg_half_elems = static_cast<int>(c->xc.half_bytes / sizeof(int32_t));
    std::memcpy(fp.bridge, c->bridge, sizeof(fp.bridge));
    fp.poll_ns = c->poll_ns;
    fp.pdl_wait = 0;
#ifdef CFGMS_TRACE
    fp.trace = c->trace_k2;
#endif
    fp.ready_target = (c->V / kBM) * kEpiWarps;   // every epilogue warp of every vocabulary tile of the stream
    if (c->use_cand) {
        size_t fsmem = static_cast<size_t>(kCandWarps) * cand_warp_words(c->V) * 4;
        const int cells = 2 * ((a->R + 1) / 2) * c->S;   // (stream, even rows | odd rows): see the kernel's cell order
        const int fblocks = (cells + kCandWarps - 1) / kCandWarps;
        // Serial mode, at most two CTAs per SM: K2 is launched as a programmatic dependent of K1 all the same —
        // it is scheduled while the GEMM runs, fetches its per-request parameters and waits on the device
        // (griddepcontrol.wait) for the GEMM's results, which hides its launch latency (config 2: 17.6 vs 18.1,
        // config 3: 69.6 vs 70.1 us/step).  A dependent grid's CTAs become resident wherever an SM has room,
        // i.e. on the few SMs the GEMM left idle or frees first, up to 16 per SM, and every cell is one latency
        // chain: so each CTA asks for enough shared memory that no SM takes more than its even share.  Larger
        // grids measured slower this way (config 4, 768 CTAs: 64.5 vs 59.0 us/step) and keep the plain launch.
        const bool pdl_k2 = !overlap && !prof && c->overlap_mode != 1 && c->pdl_finalize && fblocks <= 2 * c->num_sms;
        fp.pdl_wait = pdl_k2 ? 1 : 0;
        if (pdl_k2) {
            const int per_sm = std::max(1, (fblocks + c->num_sms - 1) / c->num_sms);
            const size_t spread = (static_cast<size_t>(c->max_smem_optin) / per_sm) & ~static_cast<size_t>(1023);
            if (spread > fsmem + 2048) fsmem = spread - 2048;
        }
        using FinFn = void (*)(const FinalizeParams);
        const FinFn ffn = c->V <= 1024 ? cfgms_finalize_cand_kernel<1> : c->V <= 2048 ? cfgms_finalize_cand_kernel<2>
                        : c->V <= 4096 ? cfgms_finalize_cand_kernel<4> : cfgms_finalize_cand_kernel<8>;
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3(static_cast<unsigned>(fblocks));
        lc.blockDim = dim3(kCandWarps * 32);
        lc.dynamicSmemBytes = fsmem;
        lc.stream = st;
        // Programmatic dependent launch: K2's CTAs are scheduled beside the still-running K1 (which
        // triggers right after its setup) and wait per cell on the ready counters.  With the profiling
        // events between the two launches the kernels run back to back instead.
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = attr;
        lc.numAttrs = ((overlap && !prof) || pdl_k2) ? 1 : 0;
        if (cudaLaunchKernelEx(&lc, ffn, fp) != cudaSuccess) {
            // K1 is already enqueued: leave no armed counters behind for the next step's K2
            if (c->ready) cudaMemsetAsync(c->ready, 0, static_cast<size_t>(c->ready_words - 32) * sizeof(int), st);
            return CFGMS_ERR_CUDA;
        }
    } else {
        const dim3 fgrid(c->S, a->R);
        const size_t fsmem = static_cast<size_t>(c->V) * 8;
        if (c->V <= 256 * 4) cfgms_finalize_kernel<4><<<fgrid, kFinThreads, fsmem, st>>>(fp);
        else if (c->V <= 256 * 8) cfgms_finalize_kernel<8><<<fgrid, kFinThreads, fsmem, st>>>(fp);
        else if (c->V <= 256 * 16) cfgms_finalize_kernel<16><<<fgrid, kFinThreads, fsmem, st>>>(fp);
        else if (c->V <= 256 * 32) cfgms_finalize_kernel<32><<<fgrid, kFinThreads, fsmem, st>>>(fp);
        else cfgms_finalize_large_kernel<<<fgrid, kFinThreads, static_cast<size_t>(c->V) * 4, st>>>(fp);
    }
    ++launches;
    if (prof) { cudaEventRecord(c->prof_ev[3 * c->prof_n + 2], st); ++c->prof_n; }

    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.row_tile = BN; c->info.row_blocks = nrb; c->info.gemm_grid = grid; c->info.pipeline_stages = stages;
    c->info.cta_pair = pair ? 1 : 0;
    c->info.split_k = split ? 2 : 1;
    c->info.overlap = (overlap && !prof) ? 1 : 0;
    c->info.launches_last_step = launches;
    c->info.launches_total += launches;
    c->info.h2d_bytes_last_step = 0; c->info.d2h_bytes_last_step = 0;
    return CFGMS_OK;
}

}  // namespace

extern "C" {

int cfgms_step(cfgms_ctx* c, const cfgms_step_args* a, void* cuda_stream) {
    const int rc = validate_step(c, a);
    if (rc != CFGMS_OK) return rc;
    return step_impl(c, a, static_cast<cudaStream_t>(cuda_stream), nullptr);
}

int cfgms_step_host(cfgms_ctx* c, const cfgms_step_args* a, void* cuda_stream) {
    int rc = validate_step(c, a);
    if (rc != CFGMS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    HostStage& h = c->hs;
    const size_t Rmax = static_cast<size_t>(c->max_rows);
    if (!c->hs_ready) {
        // every per-row input of a step travels in ONE block: nine [R] arrays (the seven of the plain path, phase and
        // phase_pos) + force_token [R][S]
        h.params_bytes = Rmax * 4 * (9 + static_cast<size_t>(c->S));
        bool ok = cudaMalloc(&h.hidden, Rmax * c->d * 4) == cudaSuccess &&
                  cudaMalloc(reinterpret_cast<void**>(&h.params), h.params_bytes) == cudaSuccess &&
                  cudaMallocHost(reinterpret_cast<void**>(&h.params_pinned), h.params_bytes) == cudaSuccess &&
                  dev_alloc(&h.tokens, Rmax * c->S) == CFGMS_OK && dev_alloc(&h.frame, Rmax * c->S) == CFGMS_OK &&
                  dev_alloc(&h.frame_index, Rmax) == CFGMS_OK &&
                  cudaStreamCreateWithFlags(&h.copy_stream, cudaStreamNonBlocking) == cudaSuccess;
        for (int j = 0; ok && j < 16; ++j) ok = cudaEventCreateWithFlags(&h.chunk_ev[j], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) {      // leave nothing half-built behind: the next call starts over
            cudaFree(h.hidden); cudaFree(h.params); cudaFreeHost(h.params_pinned);
            cudaFree(h.tokens); cudaFree(h.frame); cudaFree(h.frame_index);
            for (int j = 0; j < 16; ++j) { if (h.chunk_ev[j]) cudaEventDestroy(h.chunk_ev[j]); h.chunk_ev[j] = nullptr; }
            if (h.copy_stream) cudaStreamDestroy(h.copy_stream);
            h.hidden = nullptr; h.params = nullptr; h.params_pinned = nullptr; h.tokens = h.frame = h.frame_index = nullptr;
            h.copy_stream = nullptr;
            return CFGMS_ERR_NOMEM;
        }
        c->hs_ready = true;
    }
    const size_t R = static_cast<size_t>(a->R);
    int64_t h2d = 0;
    // pack the small arrays into the pinned mirror (a few tens of KB), one copy for all of them
    size_t off = 0;
    auto pack = [&](const void* src, size_t bytes) -> char* {
        if (!src) return nullptr;
        std::memcpy(h.params_pinned + off, src, bytes);
        char* dev = h.params + off;
        off += bytes;
        return dev;
    };
    cfgms_step_args d = *a;
    d.pair_map = reinterpret_cast<const int32_t*>(pack(a->pair_map, R * 4));
    d.w = reinterpret_cast<const float*>(pack(a->w, R * 4));
    d.temp = reinterpret_cast<const float*>(pack(a->temp, R * 4));
    d.top_k = reinterpret_cast<const int32_t*>(pack(a->top_k, R * 4));
    d.step = reinterpret_cast<const int32_t*>(pack(a->step, R * 4));
    d.req_id = reinterpret_cast<const uint32_t*>(pack(a->req_id, R * 4));
    d.n_frames = reinterpret_cast<const int32_t*>(pack(a->n_frames, R * 4));
    d.force_token = reinterpret_cast<const int32_t*>(pack(a->force_token, R * c->S * 4));
    d.phase = reinterpret_cast<const int32_t*>(pack(a->phase, R * 4));          // read by the GEMM epilogue and the samplers
    d.phase_pos = reinterpret_cast<const int32_t*>(pack(a->phase_pos, R * 4));
    if (cudaMemcpyAsync(h.params, h.params_pinned, off, cudaMemcpyHostToDevice, st) != cudaSuccess) return CFGMS_ERR_CUDA;
    h2d += static_cast<int64_t>(off);
    d.tokens_out = h.tokens;
    d.frame_out = a->frame_out ? h.frame : nullptr;
    d.frame_index_out = a->frame_index_out ? h.frame_index : nullptr;
    d.hidden = h.hidden;
    if (a->hidden_dtype == CFGMS_BF16) {
        // hidden states: uploaded in two chunks on the copy stream, each chunk's GEMM launch waits for its own
        // chunk only (step_impl).  The copy stream first waits for whatever precedes this call on the caller's stream.
        if (cudaEventRecord(h.chunk_ev[15], st) != cudaSuccess || cudaStreamWaitEvent(h.copy_stream, h.chunk_ev[15], 0) != cudaSuccess)
            return CFGMS_ERR_CUDA;
        HostUpload up{static_cast<const char*>(a->hidden), static_cast<char*>(h.hidden), &h2d};
        rc = step_impl(c, &d, st, &up);
    } else {
        const size_t hid_bytes = R * c->d * 4;
        if (cudaMemcpyAsync(h.hidden, a->hidden, hid_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return CFGMS_ERR_CUDA;
        h2d += static_cast<int64_t>(hid_bytes);
        rc = step_impl(c, &d, st, nullptr);
    }
    if (rc != CFGMS_OK) return rc;
    const size_t tok_bytes = R * c->S * 4;
    if (cudaMemcpyAsync(a->tokens_out, h.tokens, tok_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return CFGMS_ERR_CUDA;
    int64_t d2h = static_cast<int64_t>(tok_bytes);
    if (a->frame_out) {
        if (cudaMemcpyAsync(a->frame_out, h.frame, tok_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return CFGMS_ERR_CUDA;
        d2h += static_cast<int64_t>(tok_bytes);
    }
    if (a->frame_index_out) {
        if (cudaMemcpyAsync(a->frame_index_out, h.frame_index, R * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return CFGMS_ERR_CUDA;
        d2h += static_cast<int64_t>(R * 4);
    }
    if (cudaStreamSynchronize(st) != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.h2d_bytes_last_step = h2d;
    c->info.d2h_bytes_last_step = d2h;
    return CFGMS_OK;
}

int cfgms_set_logit_bias(cfgms_ctx* c, const float* bias, void* cuda_stream) {
    if (!c) return CFGMS_ERR_ARG;
    const int blocks = (c->NT + 255) / 256;
    cfgms_bias_fold_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(c->bias_base, bias, c->bias, c->NT);
    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.launches_total += 1;
    return CFGMS_OK;
}

int cfgms_set_stream_vocab_sizes(cfgms_ctx* c, const int32_t* sizes, const float* extra_bias, void* cuda_stream) {
    if (!c || !sizes) return CFGMS_ERR_ARG;
    StreamSizes sz;
    for (int i = 0; i < 64; ++i) sz.v[i] = 0;
    for (int i = 0; i < c->S; ++i) {
        if (sizes[i] < 1 || sizes[i] > c->V) return CFGMS_ERR_ARG;
        sz.v[i] = sizes[i];
    }
    const int blocks = (c->NT + 255) / 256;
    cfgms_bias_fold_ragged_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(c->bias_base, extra_bias, c->bias,
                                                                                            c->NT, c->V, sz);
    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.launches_total += 1;
    return CFGMS_OK;
}

int cfgms_exchange_create(cfgms_ctx* c, int32_t world, int32_t rank, void* ipc_handle_out, void** base_out) {
    if (!c || world < 1 || world > 64 || rank < 0 || rank >= world) return CFGMS_ERR_ARG;
    if (c->S_total == 0 || c->xc.base) return CFGMS_ERR_ARG;       // needs the global stream count; one exchange per context
    // [half 0 | half 1 | latest | flags uint32 [64] | state]: peers write the halves and the flags only
    c->xc.half_bytes = (static_cast<size_t>(c->max_rows) * c->S_total * sizeof(int32_t) + 255) & ~static_cast<size_t>(255);
    c->xc.latest_off = 2 * c->xc.half_bytes;
    c->xc.flags_off = 3 * c->xc.half_bytes;
    c->xc.state_off = c->xc.flags_off + 256;
    const size_t total = c->xc.state_off + 256;
    if (cudaMalloc(&c->xc.base, total) != cudaSuccess) { c->xc.base = nullptr; cudaGetLastError(); return CFGMS_ERR_NOMEM; }
    // a failure below leaves no half-made exchange behind: the context is as before the call and may try again
    auto undo = [&]() { cudaFree(c->xc.base); c->xc.base = nullptr; c->xc.world = 0; c->xc.rank = 0; cudaGetLastError(); return CFGMS_ERR_CUDA; };
    if (cudaMemset(c->xc.base, 0, total) != cudaSuccess) return undo();
    c->xc.world = world; c->xc.rank = rank;
    if (ipc_handle_out) {
        static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size is part of the ABI");
        cudaIpcMemHandle_t h;
        if (cudaIpcGetMemHandle(&h, c->xc.base) != cudaSuccess) return undo();
        std::memcpy(ipc_handle_out, &h, sizeof(h));
    }
    if (base_out) *base_out = c->xc.base;
    return CFGMS_OK;
}

int cfgms_exchange_connect(cfgms_ctx* c, void* const* peer_bases) {
    if (!c || !c->xc.base || !peer_bases) return CFGMS_ERR_ARG;
    const int world = c->xc.world;
    int32_t* tok[64];
    uint32_t* flg[64];
    for (int q = 0; q < world; ++q) {
        char* base = static_cast<char*>(q == c->xc.rank ? c->xc.base : peer_bases[q]);
        if (!base) return CFGMS_ERR_ARG;
        tok[q] = reinterpret_cast<int32_t*>(base);
        flg[q] = reinterpret_cast<uint32_t*>(base + c->xc.flags_off);
    }
    if (!c->xc.d_tokens && (dev_alloc(&c->xc.d_tokens, 64) != CFGMS_OK || dev_alloc(&c->xc.d_flags, 64) != CFGMS_OK)) return CFGMS_ERR_NOMEM;
    if (cudaMemcpy(c->xc.d_tokens, tok, sizeof(int32_t*) * world, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(c->xc.d_flags, flg, sizeof(uint32_t*) * world, cudaMemcpyHostToDevice) != cudaSuccess)
        return CFGMS_ERR_CUDA;
    c->xc.connected = true;
    return CFGMS_OK;
}

int cfgms_exchange_connect_ipc(cfgms_ctx* c, const void* handles) {
    if (!c || !c->xc.base || !handles) return CFGMS_ERR_ARG;
    void* bases[64] = {nullptr};
    for (int q = 0; q < c->xc.world; ++q) {
        if (q == c->xc.rank) continue;
        if (!c->xc.opened[q]) {
            cudaIpcMemHandle_t h;
            std::memcpy(&h, static_cast<const char*>(handles) + 64 * q, sizeof(h));
            // fails (ERR_CUDA, nothing connected) when the handle is not a live allocation of another process or the two
            // devices cannot reach each other: no peer access, no exchange
            if (cudaIpcOpenMemHandle(&c->xc.opened[q], h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
                c->xc.opened[q] = nullptr;
                cudaGetLastError();
                return CFGMS_ERR_CUDA;
            }
            // lazy peer enabling defers the real check to first use: ask now, so that a pair of GPUs without a peer path
            // is refused here and not by a faulting store inside the finalize kernel
            cudaPointerAttributes pa{};
            int can = 1;
            if (cudaPointerGetAttributes(&pa, c->xc.opened[q]) == cudaSuccess && pa.device != c->device)
                if (cudaDeviceCanAccessPeer(&can, c->device, pa.device) != cudaSuccess) { can = 1; cudaGetLastError(); }
            if (!can) {
                cudaIpcCloseMemHandle(c->xc.opened[q]);
                c->xc.opened[q] = nullptr;
                return CFGMS_ERR_CUDA;
            }
        }
        bases[q] = c->xc.opened[q];
    }
    return cfgms_exchange_connect(c, bases);
}

int cfgms_exchange_wait(cfgms_ctx* c, int32_t R, void* cuda_stream) {
    if (!c || !c->xc.connected || R < 1 || R > c->max_rows) return CFGMS_ERR_ARG;
    char* base = static_cast<char*>(c->xc.base);
    cfgms_exchange_wait_kernel<<<1, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        reinterpret_cast<const volatile uint32_t*>(base + c->xc.flags_off),
        reinterpret_cast<unsigned int*>(base + c->xc.state_off) + 2, c->xc.world,
        reinterpret_cast<const int32_t*>(base), reinterpret_cast<int32_t*>(base + c->xc.latest_off),
        static_cast<int>(c->xc.half_bytes / sizeof(int32_t)), R * c->S_total, c->err);
    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.launches_total += 1;
    return CFGMS_OK;
}

int cfgms_exchange_tokens(cfgms_ctx* c, const int32_t** tokens_all_out) {
    if (!c || !c->xc.base || !tokens_all_out) return CFGMS_ERR_ARG;
    *tokens_all_out = reinterpret_cast<const int32_t*>(static_cast<char*>(c->xc.base) + c->xc.latest_off);
    return CFGMS_OK;
}

int cfgms_set_phase_table(cfgms_ctx* c, int32_t V_text, const int32_t* bridge_tokens, int32_t n_bridge) {
    if (!c || V_text < 0 || V_text > c->V || n_bridge < 0 || n_bridge > 16 || (n_bridge > 0 && !bridge_tokens)) return CFGMS_ERR_ARG;
    // on the candidate path a vocabulary region must be whole 32-token chunks
    if (c->use_cand && (V_text % 32) != 0) return CFGMS_ERR_SHAPE;
    c->V_text = V_text;
    c->n_bridge = n_bridge;
    for (int j = 0; j < 16; ++j) c->bridge[j] = j < n_bridge ? bridge_tokens[j] : 0;
    return CFGMS_OK;
}

int cfgms_feedback(cfgms_ctx* c, const int32_t* tokens, const void* emb, int32_t V_e, int32_t R, void* x_out,
                   void* cuda_stream) {
    if (!c || R < 0 || V_e < 1) return CFGMS_ERR_ARG;
    if (R == 0) return CFGMS_OK;
    if (!tokens || !emb || !x_out) return CFGMS_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(emb) & 15u) != 0 || (reinterpret_cast<uintptr_t>(x_out) & 15u) != 0) return CFGMS_ERR_ARG;
    cfgms_feedback_kernel<<<(R + 1) / 2, kFbThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        tokens, static_cast<const __nv_bfloat16*>(emb), static_cast<__nv_bfloat16*>(x_out), R, c->S, V_e, c->d);
    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.launches_total += 1;
    return CFGMS_OK;
}

int cfgms_deinterleave(cfgms_ctx* c, const int32_t* delayed, int32_t n, int32_t T, int32_t S, int32_t* grid_out,
                       void* cuda_stream) {
    if (!c || n < 0 || S < 1 || T < S) return CFGMS_ERR_ARG;
    if (n == 0) return CFGMS_OK;
    if (!delayed || !grid_out) return CFGMS_ERR_ARG;
    if (S > 64 || n > 65535) return CFGMS_ERR_SHAPE;
    if ((reinterpret_cast<uintptr_t>(delayed) & 15u) != 0 || (reinterpret_cast<uintptr_t>(grid_out) & 15u) != 0)
        return CFGMS_ERR_ARG;
    const int F = T - S + 1;
    const dim3 grid((F + kDeintFrames - 1) / kDeintFrames, n);
    const size_t smem = static_cast<size_t>(kDeintFrames + S - 1) * S * 4;
    cfgms_deinterleave_kernel<<<grid, kDeintThreads, smem, static_cast<cudaStream_t>(cuda_stream)>>>(delayed, grid_out, T, S);
    if (cudaPeekAtLastError() != cudaSuccess) return CFGMS_ERR_CUDA;
    c->info.launches_total += 1;
    return CFGMS_OK;
}

int cfgms_deinterleave_host(cfgms_ctx* c, const int32_t* delayed, int32_t n, int32_t T, int32_t S, int32_t* grid_out,
                            void* cuda_stream) {
    if (!c || n < 0 || S < 1 || T < S) return CFGMS_ERR_ARG;
    if (n == 0) return CFGMS_OK;
    if (!delayed || !grid_out) return CFGMS_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    HostStage& h = c->hs;
    const size_t in_bytes = static_cast<size_t>(n) * T * S * 4;
    const size_t out_bytes = static_cast<size_t>(n) * (T - S + 1) * S * 4;
    if (in_bytes > h.deint_in_bytes) {
        cudaFree(h.deint_in);
        h.deint_in = nullptr; h.deint_in_bytes = 0;
        if (cudaMalloc(reinterpret_cast<void**>(&h.deint_in), in_bytes) != cudaSuccess) return CFGMS_ERR_NOMEM;
        h.deint_in_bytes = in_bytes;
    }
    if (out_bytes > h.deint_out_bytes) {
        cudaFree(h.deint_out);
        h.deint_out = nullptr; h.deint_out_bytes = 0;
        if (cudaMalloc(reinterpret_cast<void**>(&h.deint_out), out_bytes) != cudaSuccess) return CFGMS_ERR_NOMEM;
        h.deint_out_bytes = out_bytes;
    }
    if (cudaMemcpyAsync(h.deint_in, delayed, in_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return CFGMS_ERR_CUDA;
    int rc = cfgms_deinterleave(c, h.deint_in, n, T, S, h.deint_out, cuda_stream);
    if (rc != CFGMS_OK) return rc;
    if (cudaMemcpyAsync(grid_out, h.deint_out, out_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return CFGMS_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return CFGMS_ERR_CUDA;
    return CFGMS_OK;
}

int cfgms_last_device_error(cfgms_ctx* c, int32_t* row_out) {
    if (!c) return CFGMS_ERR_ARG;
    int word[2] = {0, 0};
    cudaError_t e = cudaMemcpy(word, c->err, sizeof(word), cudaMemcpyDeviceToHost);
    if (row_out) *row_out = -1;
    if (e != cudaSuccess) return CFGMS_ERR_CUDA;
    if (word[0] == 0) return CFGMS_OK;
    if (row_out) *row_out = word[0] >> 8;
    cudaMemset(c->err, 0, sizeof(word));
    if (c->ready) cudaMemset(c->ready, 0, static_cast<size_t>(c->ready_words - 32) * sizeof(int));   // a failed step may leave them armed
    return word[0] & 0xff;
}

int cfgms_profile_enable(cfgms_ctx* c, int on) {
    if (!c) return CFGMS_ERR_ARG;
    if (on && !c->prof_ev) {
        cudaEvent_t* ev = new (std::nothrow) cudaEvent_t[3 * kProfMax]();    // value-initialised: null handles
        if (!ev) return CFGMS_ERR_NOMEM;
        for (int j = 0; j < 3 * kProfMax; ++j) {
            if (cudaEventCreate(&ev[j]) != cudaSuccess) {
                for (int q = 0; q < j; ++q) cudaEventDestroy(ev[q]);
                delete[] ev;
                return CFGMS_ERR_CUDA;
            }
        }
        c->prof_ev = ev;
    }
    c->prof_on = on != 0;
    c->prof_n = 0;
    return CFGMS_OK;
}

int cfgms_profile_read(cfgms_ctx* c, double* gemm_ms, double* finalize_ms, int64_t* steps) {
    if (!c || !gemm_ms || !finalize_ms || !steps) return CFGMS_ERR_ARG;
    double g = 0.0, f = 0.0;
    for (int j = 0; j < c->prof_n; ++j) {
        float a = 0.f, b = 0.f;
        if (cudaEventSynchronize(c->prof_ev[3 * j + 2]) != cudaSuccess) return CFGMS_ERR_CUDA;
        if (cudaEventElapsedTime(&a, c->prof_ev[3 * j], c->prof_ev[3 * j + 1]) != cudaSuccess ||
            cudaEventElapsedTime(&b, c->prof_ev[3 * j + 1], c->prof_ev[3 * j + 2]) != cudaSuccess)
            return CFGMS_ERR_CUDA;
        g += a;
        f += b;
    }
    *gemm_ms = g; *finalize_ms = f; *steps = c->prof_n;
    c->prof_n = 0;
    return CFGMS_OK;
}

int cfgms_overlap_stats(cfgms_ctx* c, int64_t* cells_waited) {
    if (!c || !cells_waited) return CFGMS_ERR_ARG;
    *cells_waited = 0;
    if (!c->ready) return CFGMS_OK;
    unsigned long long w[16];
    int* st = c->ready + (c->ready_words - 32);
    if (cudaMemcpy(w, st, sizeof(w), cudaMemcpyDeviceToHost) != cudaSuccess) return CFGMS_ERR_CUDA;
    if (cudaMemset(st, 0, sizeof(w)) != cudaSuccess) return CFGMS_ERR_CUDA;
    for (int j = 0; j < 16; ++j) *cells_waited += static_cast<int64_t>(w[j]);
    return CFGMS_OK;
}

#ifdef CFGMS_TRACE
// developer build only: device buffers of 16 x u64 per CTA that K1 / K2 fill with their timeline marks
int cfgms_debug_trace(cfgms_ctx* c, unsigned long long* k1, unsigned long long* k2) {
    if (!c) return CFGMS_ERR_ARG;
    c->trace_k1 = k1; c->trace_k2 = k2;
    return CFGMS_OK;
}
#endif

int cfgms_get_info(cfgms_ctx* c, cfgms_info* out) {
    if (!c || !out) return CFGMS_ERR_ARG;
    *out = c->info;
    return CFGMS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// cfgms_deinterleave_host_static: the de-interleave with host buffers for callers that must not allocate device
// memory (a serving engine that gave all free HBM to its cache pool, a decode loop that cannot afford cudaMalloc's
// device-wide synchronisation, a deployment with a fixed memory budget; include/cfgms.h has the full contract).
// Nothing below calls cudaMalloc / cudaFree / cudaMallocHost or creates streams or events.
//
// The staging the kernel reads from and writes to is this file-scope array.  It is part of the library's device
// image: each GPU this process runs libcfgms.so on holds these 8 MiB until the process exits.  In HOST code the
// name g_static_scratch is only a handle for the runtime's symbol table, NOT a device address — handing it to a
// kernel would make the kernel fault (or, where the GPU can reach host memory, scribble over the host-side shadow).
// The device address is fetched once per device with cudaGetSymbolAddress and that pointer is what the kernel gets.
static __device__ __align__(256) unsigned char g_static_scratch[CFGMS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticScratchDevice {
    bool ready = false;
    unsigned char* base = nullptr;     // device address of g_static_scratch on this device
};
StaticScratchDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

// Once per device, with that device current: architecture check, the array's device address, and the shared-memory
// opt-in the kernel needs from S = 42 on (cfgms_create does the same for contexts; this entry point has none).
int static_scratch_setup(unsigned char** base_out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CFGMS_ERR_CUDA; }
    if (dev < 0 || dev >= kStaticMaxDevices) return CFGMS_ERR_ARG;
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticScratchDevice& sd = g_static_dev[dev];
    if (!sd.ready) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return CFGMS_ERR_CUDA; }
        if (major != 10) return CFGMS_ERR_ARCH;
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return CFGMS_ERR_CUDA; }
        if (cudaFuncSetAttribute(cfgms_deinterleave_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024) != cudaSuccess) {
            cudaGetLastError();
            return CFGMS_ERR_CUDA;
        }
        sd.base = static_cast<unsigned char*>(p);
        sd.ready = true;
    }
    *base_out = sd.base;
    return CFGMS_OK;
}

}  // namespace

extern "C" int cfgms_deinterleave_host_static(const int32_t* delayed, int32_t n, int32_t T, int32_t S, int32_t* grid_out,
                                              void* cuda_stream) {
    if (n < 0 || S < 1 || T < S) return CFGMS_ERR_ARG;
    if (n == 0) return CFGMS_OK;
    if (!delayed || !grid_out) return CFGMS_ERR_ARG;
    if (S > 64 || n > 65535) return CFGMS_ERR_SHAPE;
    const int F = T - S + 1;
    const size_t in_bytes = static_cast<size_t>(n) * static_cast<size_t>(T) * S * 4;
    const size_t out_bytes = static_cast<size_t>(n) * static_cast<size_t>(F) * S * 4;
    const size_t out_off = (in_bytes + 255) & ~static_cast<size_t>(255);      // both halves 256-byte aligned (the kernel needs 16)
    if (out_off + out_bytes > static_cast<size_t>(CFGMS_STATIC_SCRATCH_BYTES)) return CFGMS_ERR_LIMIT;

    unsigned char* base = nullptr;
    const int rc = static_scratch_setup(&base);
    if (rc != CFGMS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int32_t* d_in = reinterpret_cast<int32_t*>(base);
    int32_t* d_out = reinterpret_cast<int32_t*>(base + out_off);
    // The array still holds the previous call's bytes.  That is harmless: the kernel reads d_in[0, n*T*S) only, all of
    // it uploaded just now, and writes every word of d_out[0, n*F*S), which is all that is copied back.
    if (cudaMemcpyAsync(d_in, delayed, in_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaGetLastError(); return CFGMS_ERR_CUDA; }
    const dim3 grid((F + kDeintFrames - 1) / kDeintFrames, n);
    const size_t smem = static_cast<size_t>(kDeintFrames + S - 1) * S * 4;
    cfgms_deinterleave_kernel<<<grid, kDeintThreads, smem, st>>>(d_in, d_out, T, S);
    if (cudaGetLastError() != cudaSuccess) { cudaStreamSynchronize(st); return CFGMS_ERR_CUDA; }
    if (cudaMemcpyAsync(grid_out, d_out, out_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) { cudaGetLastError(); cudaStreamSynchronize(st); return CFGMS_ERR_CUDA; }
    if (cudaStreamSynchronize(st) != cudaSuccess) return CFGMS_ERR_CUDA;
    return CFGMS_OK;
}
