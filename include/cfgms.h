/*
 * cfgms.h — C ABI of the B200-native CFG multi-stream audio decode head.
 *
 * One library call = one step of the per-step audio decode head of the SpeechLM serving
 * pipeline of arxiv 2607.02119 (citations: PAPER.md line numbers), for a continuous batch in
 * which every classifier-free-guidance (CFG) conditional row sits next to its unconditional
 * companion (Paired Request Co-Scheduling):
 *
 *   1. head projection      l^(i) = W_H (h_t + e_i), i = 0..S-1
 *   2. CFG merge            l~ = w l_cond + (1 - w) l_uncond   (Eq. 1)
 *   3. sampling             temperature, top-k, Gumbel-max over Philox4x32-10 noise keyed by
 *                           (seed, request, step, stream, token)
 *   4. token sync + delay   same token to the companion row; delayed[row][tau][i] with
 *                           stream i lagging i steps; PAD outside the frame range
 *                                                                          PAPER.md:56,66,76,93
 *   5. de-interleave        grid[q][f][i] = delayed[q][f + i][i]
 *
 * Everything runs in hand-written sm_100a kernels; there is no CPU fallback: cfgms_create
 * returns CFGMS_ERR_ARCH on any other device.  All entry points return a cfgms_status, never
 * abort and never throw.  cfgms_step and cfgms_deinterleave only enqueue work on the given
 * stream and never synchronise (they are CUDA-graph capturable); the *_host variants copy
 * through library-owned device staging and synchronise the stream before returning.
 *
 * Ownership: the library owns only what it allocates (bias, scratch logits, staging, error
 * word).  Every user pointer is borrowed; `heads` must stay valid for the context lifetime.
 */
#ifndef CFGMS_H
#define CFGMS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cfgms_ctx cfgms_ctx; /* opaque */

typedef enum {
    CFGMS_OK = 0,
    CFGMS_ERR_ARG = 1,    /* null pointer, non-positive size, bad enum                         */
    CFGMS_ERR_SHAPE = 2,  /* d % 8 != 0, S > 64, R > max_rows, V too large for the sampler ... */
    CFGMS_ERR_LAYOUT = 3, /* pair_map contract violated (reported by cfgms_last_device_error)  */
    CFGMS_ERR_CUDA = 4,   /* a CUDA runtime / driver call failed                               */
    CFGMS_ERR_ARCH = 5,   /* device is not compute capability 10.x                             */
    CFGMS_ERR_NOMEM = 6,
    CFGMS_ERR_TIMEOUT = 7, /* a device-side pipeline wait gave up (reported asynchronously)    */
    CFGMS_ERR_LIMIT = 8   /* the request needs more than the fixed scratch of an entry point that
                             never allocates (cfgms_deinterleave_host_static)                  */
} cfgms_status;

typedef enum { CFGMS_BF16 = 0, CFGMS_F32 = 1 } cfgms_dtype;

/* cfgms_config.flags */
#define CFGMS_CFG_PAD_TOKEN 1u /* use cfgms_config.pad_token instead of the default (= V)      */
#define CFGMS_CFG_NO_CANDIDATES 2u /* tuning/debug: never use the fused per-chunk candidate pass;
                                      the sampler then scans all V logits of every cell (the path
                                      always taken when V % 32 != 0 or V > 8192)                 */

#define CFGMS_CFG_SINGLE_CTA 4u  /* tuning/debug: never pair CTAs on one M = 256 MMA                */
#define CFGMS_CFG_CTA_PAIR 8u    /* tuning/debug: always run the head GEMM on CTA pairs (cta_group::2) */
#define CFGMS_CFG_NO_OVERLAP 16u /* tuning/debug: always launch the finalize kernel strictly after the
                                    head GEMM.  Default: when the GEMM runs several waves of tiles, the
                                    finalize kernel is launched as its programmatic dependent and samples
                                    finished (stream, row block) groups while the GEMM is still running
                                    (candidate path with V % 128 == 0)                                 */
#define CFGMS_CFG_OVERLAP 32u    /* tuning/debug: overlap whenever eligible, even for a one-wave GEMM   */

#define CFGMS_CFG_NO_PDL_FINALIZE 64u /* tuning/debug: always launch the finalize kernel as an ordinary stream-ordered
                                    kernel.  Default for small finalize grids that do not overlap the GEMM
                                    through the ready counters: programmatic dependent launch — scheduled while
                                    the GEMM runs, it fetches its per-request parameters and waits on the device
                                    (griddepcontrol.wait) for the GEMM's results                          */

#define CFGMS_CFG_NO_SPLIT_K 128u /* tuning/debug: never run a one-wave head GEMM as split-K clusters of four CTAs
                                    (two CTA pairs that each stream half of K and exchange partial sums over
                                    distributed shared memory; the default whenever the (vocabulary tile pair,
                                    128-row block) tiles fill at most a quarter of the SMs)                   */

typedef struct {
    int32_t max_rows;  /* largest R accepted by cfgms_step; <= 0 means 1024                     */
    int32_t pad_token; /* written at inactive (step, stream) cells when CFGMS_CFG_PAD_TOKEN      */
    uint32_t flags;
    int32_t row_tile;  /* debug/tuning: batch rows per accumulator tile (multiple of 64,
                          <= 256); 0 = chosen from R and the SM count                           */
    int32_t max_stages; /* debug/tuning: cap on the head GEMM's TMA ring depth (0 = as deep as fits)   */
    int32_t stream_base;   /* stream-sharded heads (one context per GPU, each holding some of the     */
    int32_t stream_stride; /* streams): local stream i of THIS context is global stream
                              stream_base + i * stream_stride.  The delay pattern, the noise key and
                              the primary-stream rules use the global index, so the shards together
                              sample exactly what one unsharded context samples; the caller gathers
                              tokens_out [R][S_local] of all shards (<= 32 KB per step).  stride <= 0
                              means unsharded (base 0, stride 1).  frame_out needs an unsharded context */
    int32_t global_streams; /* stream-sharded heads: the number of streams of the WHOLE head (the drain of a
                               request ends S_global - 1 steps after its last frame); 0 = this context's S.
                               A sharded context needs it to write step_next_out / n_frames_next_out / done_out.
                               Only the shard that holds global stream 0 (stream_base == 0) can write the request-state
                               outputs (step_next_out, n_frames_next_out, done_out, phase_next_out, phase_pos_next_out,
                               modality_out): the state advances on the primary stream's token.  Any other shard that
                               asks for them gets CFGMS_ERR_ARG; it takes the next state from the rank with stream 0
                               (4 small [R] arrays) or keeps passing host-advanced state                         */
} cfgms_config;

/*
 * cfgms_create — PAPER.md:54 (shared head W_H over S audio sub-vocabularies, stream
 * embeddings e_i).  Builds bias[i][v] = sum_k W_i[v][k] e_i[k] once (fp32), so that the
 * per-step contraction runs on h_t alone and e_i is never rounded into bf16 with it.
 *   heads  : DEVICE, bf16 [S][V][d], k contiguous. BORROWED for the context lifetime.
 *   embeds : DEVICE, bf16 [S][d]. Read during the call only.
 *   S, d, V: streams, hidden width, tokens per codebook. Requires d % 8 == 0, 1 <= S <= 64.
 *   cfg    : nullable.
 * Synchronises the device once.  Errors: ARG, SHAPE, ARCH, NOMEM, CUDA.
 */
int cfgms_create(cfgms_ctx** out, const void* heads, const void* embeds, int32_t S, int32_t d,
                 int32_t V, const cfgms_config* cfg);
void cfgms_destroy(cfgms_ctx* ctx);

/*
 * Arguments of one decode step.  Arrays are indexed by batch row r in [0, R).
 * Batch layout contract (the product of paired co-scheduling): the batch is a
 * sequence of two-row slots; a slot holds one (cond, uncond) pair — cond on the EVEN row c,
 * pair_map[c] = c + 1, pair_map[c + 1] = c — or two unpaired rows with pair_map = -1.
 * Per-request values (w, temp, top_k, step, req_id, n_frames) are read at the cond row of a
 * pair or at the unpaired row; the companion row's entries are ignored.
 */
typedef struct {
    const void* hidden;       /* [R][d] backbone hidden states h_t, dtype below                  */
    int32_t hidden_dtype;     /* cfgms_dtype; CFGMS_F32 is rounded to bf16 (RNE) first           */
    int32_t R;                /* rows in the batch, 1 <= R <= max_rows                           */
    const int32_t* pair_map;  /* [R]                                                             */
    const float* w;           /* [R] CFG scale of Eq. 1 (any finite value)                       */
    const float* temp;        /* [R] temperature; 0 => greedy argmax                             */
    const int32_t* top_k;     /* [R] <= 0 or >= V: no filter; 1: greedy; ties at the k-th value
                                 are all kept (threshold semantics)                              */
    uint64_t seed;            /* Philox key                                                      */
    const int32_t* step;      /* [R] request-local decode step tau >= 0: keys the noise and the
                                 delay pattern (stream i active iff i <= tau < n_frames + i)     */
    const uint32_t* req_id;   /* [R] request identity for the noise; NULL => the row index       */
    const int32_t* n_frames;  /* [R] frames F of the request; NULL => no drain phase             */
    int32_t* tokens_out;      /* [R][S] sampled tokens; the companion row receives a copy        */
    int32_t* delayed;         /* nullable [R][T_cap][S] delayed-layout buffer, indexed by the
                                 cond / unpaired batch row; cell [r][tau mod T_cap][i] is written */
    int32_t T_cap;
    float* logits_out;        /* nullable DEBUG tap: merged pre-temperature logits fp32
                                 [R][S][V], valid at cond / unpaired rows                        */
    /* --- widenings (all nullable; NULL leaves the step exactly as described above) --- */
    const int32_t* force_token; /* [R][S], read at the cond / unpaired row: a value >= 0 is emitted
                                 as that cell's token without sampling — the hook for the phase
                                 state machine's deterministic bridging tokens and text-phase
                                 padding; < 0 = sample.  Only consulted for cells
                                 the delay pattern leaves active (PAD wins otherwise)            */
    int32_t* frame_out;       /* [R][S] streaming frame emission: when frame
                                 f = tau - S + 1 of the request completes at this step
                                 (0 <= f < n_frames), frame_out[r][i] = delayed[r][(f+i) mod T_cap][i];
                                 otherwise the row is filled with the pad token.  Needs `delayed`
                                 with T_cap >= S (else CFGMS_ERR_ARG).  Companion rows: pad      */
    int32_t* frame_index_out; /* [R] the frame index f emitted for the row, or -1 (also -1 at
                                 companion rows, whose outputs stay hidden)         */
    /* device-resident request state with automatic drain.  With these three the
       decode loop needs no host bookkeeping: feed step_next_out / n_frames_next_out of one step
       as step / n_frames of the next (two buffers, alternating).  Written at cond / unpaired rows. */
    int32_t eos_token;        /* end-of-audio id on the PRIMARY stream (stream 0); < 0 = none.  When
                                 stream 0 emits it at step tau while the request's frame count is
                                 still CFGMS_FRAMES_UNSET, the frame count becomes tau: stream 0
                                 pads from the next step on, stream i keeps sampling i more steps  */
    int32_t* step_next_out;   /* [R] tau + 1                                                       */
    int32_t* n_frames_next_out; /* [R] the frame count after this step (CFGMS_FRAMES_UNSET until the
                                 end-of-audio token appears; n_frames == NULL reads as UNSET)       */
    int32_t* done_out;        /* [R] 1 when the request is fully drained after this step
                                 (tau + 1 >= frames + S - 1), else 0                               */
    /* per-request phase state machine on the device; see cfgms_set_phase_table.
       phase == NULL: every request is in the audio phase with audio-local step = step[r] (the plain path). */
    const int32_t* phase;     /* [R] cfgms_phase of the request, read at the cond / unpaired row              */
    const int32_t* phase_pos; /* [R] TRANSITION: bridging tokens emitted so far; AUDIO: the audio-local step
                                 tau_a (delay pattern, frame count, ring slot); ignored otherwise.  With
                                 phases, step[r] is the request's GLOBAL step and only keys the noise, and
                                 n_frames counts audio-local steps.  Required when `phase` is given; force_token
                                 must then be NULL (the transition phase is the forced-token mechanism)  */
    int32_t* phase_next_out;  /* [R] nullable: the phase after this step                                    */
    int32_t* phase_pos_next_out; /* [R] nullable: phase_pos after this step.  Feed both back as phase / phase_pos
                                 (two buffers, alternating), together with step_next_out / n_frames_next_out  */
    int32_t* modality_out;    /* [R] nullable: 1 when a TEXT-phase request's unmasked stream-0 logits peak in the
                                 audio region (the inference that ends its text phase), else 0                */
} cfgms_step_args;

/* Phases of a request.  The PRIMARY stream (global stream 0) carries text: its V logits cover
 * the disjoint regions [0, V_text) = text tokens and [V_text, V) = its audio codes (and the end-of-audio id);
 * the other streams are audio only.  "Dynamic vocabulary masking" = the phase selects the region sampled from.
 *   TEXT        only stream 0 samples, from the text region, from the CONDITIONAL row's logits alone (the CFG
 *               merge "operates only during the audio phase"); the other streams emit the pad
 *               token.  The modality the model asks for is the region of the argmax of stream 0's unmasked
 *               logits; when it is the audio region the request moves on after this step.
 *   TRANSITION  stream 0 emits the deterministic bridging tokens, one per step; nothing is sampled.
 *   AUDIO       the hot path as described above with the audio-local step tau_a = phase_pos; stream 0 is
 *               restricted to its audio region; the end-of-audio token (eos_token) on stream 0 fixes the frame
 *               count and the drain runs S - 1 more steps; then
 *   DONE        every stream emits the pad token, the state is frozen, done_out = 1.                        */
typedef enum { CFGMS_PHASE_TEXT = 0, CFGMS_PHASE_TRANSITION = 1, CFGMS_PHASE_AUDIO = 2, CFGMS_PHASE_DONE = 3 } cfgms_phase;

#define CFGMS_FRAMES_UNSET 2147483647 /* n_frames value meaning "no frame count yet" (no drain)   */

/*
 * One step in flight per context: the merged-logit spill, the candidate lists and the ready counters are
 * the context's, so calls on one context must be enqueued on one stream (or otherwise ordered); use one
 * context per concurrent stream.  Contexts are not thread-safe; distinct contexts are independent.
 *
 * cfgms_step — steps 1-4 above for one batch.  Every pointer in `args` is a DEVICE pointer.
 * Enqueues on `cuda_stream` (a cudaStream_t, may be NULL for the default stream); does not
 * synchronise.  Errors detected on the host: ARG, SHAPE, CUDA.  A violated pair_map contract
 * or a pipeline time-out is detected on the device and latched in a sticky error word
 * (cfgms_last_device_error); the offending slot's tokens are then unspecified.
 */
int cfgms_step(cfgms_ctx* ctx, const cfgms_step_args* args, void* cuda_stream);

/*
 * cfgms_step_host — same step with HOST buffers: hidden, pair_map, w, temp, top_k, step,
 * req_id, n_frames, force_token, phase, phase_pos, tokens_out, frame_out and frame_index_out are HOST pointers
 * (pinned memory recommended); `delayed`, `logits_out` and the request-state outputs (`step_next_out`,
 * `n_frames_next_out`, `done_out`, `phase_next_out`, `phase_pos_next_out`, `modality_out`) stay DEVICE pointers
 * (per-request state lives in HBM) or NULL.  Every INPUT of this entry point is a host array, every state OUTPUT a
 * device array: a caller that keeps the phase state on the device uses cfgms_step.  Copies the
 * inputs host->device, runs the step, copies tokens_out device->host and synchronises the
 * stream.  Bytes moved per call are reported by cfgms_get_info.
 */
int cfgms_step_host(cfgms_ctx* ctx, const cfgms_step_args* args, void* cuda_stream);

/*
 * cfgms_set_logit_bias — dynamic vocabulary masking hook.  bias: DEVICE fp32
 * [S][V] added to the merged logits of every request before the temperature (-inf removes a
 * token from stream i's vocabulary), or NULL to clear it.  Folded into the library's own
 * per-token bias once, on `cuda_stream`; costs nothing per step.  Not retained.
 */
int cfgms_set_logit_bias(cfgms_ctx* ctx, const float* bias, void* cuda_stream);

/*
 * cfgms_set_phase_table — configuration of the phase state machine: V_text = size of the text
 * region of stream 0 (0 <= V_text <= V; a multiple of 32 when V is, so that a region is whole candidate chunks),
 * bridge_tokens = HOST int32 [n_bridge], 0 <= n_bridge <= 16, the deterministic bridging tokens of the
 * transition phase (copied).  Takes effect for steps enqueued afterwards.  Errors: ARG, SHAPE.
 */
int cfgms_set_phase_table(cfgms_ctx* ctx, int32_t V_text, const int32_t* bridge_tokens, int32_t n_bridge);

/*
 * cfgms_set_stream_vocab_sizes — ragged per-stream vocabularies on the uniform [S][V][d] layout (PAPER.md:104-105:
 * OpusLM's SSL stream and codec streams differ in size): stream i only ever samples tokens < sizes[i].
 * sizes: HOST int32 [S], 1 <= sizes[i] <= V; extra_bias: DEVICE fp32 [S][V] additive bias applied as well, or
 * NULL.  Replaces whatever cfgms_set_logit_bias installed (same mechanism: folded once into the per-token bias
 * of the GEMM epilogue, -inf on the padded tail).  Errors: ARG.
 */
int cfgms_set_stream_vocab_sizes(cfgms_ctx* ctx, const int32_t* sizes, const float* extra_bias, void* cuda_stream);

/*
 * Stream-sharded heads: the token exchange as a device-side operation (decode is memory-bound,
 * so dividing the weight stream over G GPUs is the lever; the heads are per stream).  Every rank g
 * creates its context with stream_base = g, stream_stride = G, global_streams = S_global and sees all rows; the
 * step's one exchange is an all-gather of the sampled tokens, done BY THE FINALIZE KERNEL: the thread that
 * writes a cell's token also stores it into every rank's gather buffer int32 [max_rows][S_global] (peer-mapped
 * memory, NVLink), and the grid's last CTA then raises one flag per destination.  No collective library call is
 * on the data path.  The gather buffer is double-buffered by step parity: a rank can run at most one step ahead of
 * a peer (its next step needs that peer's tokens), so the half it overwrites has been consumed everywhere.
 *   cfgms_exchange_create       allocates this rank's block (gather buffer + flags) with cudaMalloc; returns its
 *                               CUDA IPC handle (64 bytes, nullable) and/or its device address (nullable).  All ranks
 *                               must use the same max_rows and S_global.
 *   cfgms_exchange_connect      peer_bases: HOST array [world] of the ranks' block addresses AS VALID IN THIS
 *                               PROCESS (entry [rank] is ignored): for peers in the same process or memory
 *                               mapped by other means; from then on every cfgms_step of this context scatters.
 *   cfgms_exchange_connect_ipc  handles: HOST [world][64] bytes, every rank's IPC handle in rank order; opens the
 *                               peers' blocks (closed at cfgms_destroy) and connects.
 *   cfgms_exchange_wait         enqueues a one-CTA kernel that waits (bounded, 2 s) until the
 *                               tokens of every rank's current step have landed in this rank's gather buffer, then
 *                               copies rows [0, R) of the step's half to the buffer cfgms_exchange_tokens returns;
 *                               kernels enqueued after it on the stream may read that.  Call it exactly once per
 *                               step.  Epochs are counted on the device: CUDA-graph replay is fine.
 *   cfgms_exchange_tokens       *tokens_all_out = the gathered tokens of the last waited step, DEVICE int32
 *                               [max_rows][S_global] (owned by the context).
 * A wait that gives up after 2 s latches CFGMS_ERR_TIMEOUT in the sticky error word (cfgms_last_device_error) and
 * ends the kernel WITHOUT touching the gathered tokens or the step count (the CUDA context stays usable; whatever
 * the stream runs next reads the previous step's tokens, so check the error word before trusting a step that may
 * have met a late peer, e.g. the very first one).  A failed cfgms_exchange_create leaves no exchange behind and may
 * be repeated.  Teardown: peers store into this rank's block until their last step has finished, so synchronise
 * every rank's stream and pass a barrier of your own (host side) BEFORE any rank calls cfgms_destroy.
 * Status: the cross-process path (IPC handles, two GPUs) has not yet been run on hardware — no multi-GPU box was
 * available; the protocol is covered on one GPU (contexts of one process) and by a two-process host model.
 * Errors: ARG (no global stream count, exchange already created / not created), NOMEM, CUDA.
 */
int cfgms_exchange_create(cfgms_ctx* ctx, int32_t world, int32_t rank, void* ipc_handle_out, void** base_out);
int cfgms_exchange_connect(cfgms_ctx* ctx, void* const* peer_bases);
int cfgms_exchange_connect_ipc(cfgms_ctx* ctx, const void* handles);
int cfgms_exchange_wait(cfgms_ctx* ctx, int32_t R, void* cuda_stream);
int cfgms_exchange_tokens(cfgms_ctx* ctx, const int32_t** tokens_all_out);

/*
 * cfgms_feedback — autoregressive feedback aggregation ("the input representation
 * at each step aggregates the embeddings of these previously generated tokens"):
 *     x_out[r][k] = bf16_rne( sum_{i < S} emb[i][tokens[r][i]][k] )     (fp32 sum, i ascending)
 *   tokens : DEVICE int32 [R][S] (cfgms_step's tokens_out: a companion row carries its cond
 *            row's tokens, so both get the same input row)
 *   emb    : DEVICE bf16 [S][V_e][d] token-embedding tables, one per stream; a token id outside
 *            [0, V_e) (e.g. a pad id with no embedding row) contributes nothing
 *   x_out  : DEVICE bf16 [R][d]
 * S and d are the context's.  Enqueues on `cuda_stream`; does not synchronise.  Errors: ARG.
 */
int cfgms_feedback(cfgms_ctx* ctx, const int32_t* tokens, const void* emb, int32_t V_e, int32_t R,
                   void* x_out, void* cuda_stream);

/*
 * cfgms_deinterleave — PAPER.md:56,68: grid[q][f][i] = delayed[q][f + i][i] for
 * 0 <= f < T - S + 1.  delayed: DEVICE int32 [n][T][S]; grid_out: DEVICE int32
 * [n][T - S + 1][S].  Requires T >= S >= 1; n == 0 is a no-op.  Does not synchronise.
 */
int cfgms_deinterleave(cfgms_ctx* ctx, const int32_t* delayed, int32_t n, int32_t T, int32_t S,
                       int32_t* grid_out, void* cuda_stream);
/* Same with HOST buffers (copies in, runs, copies out, synchronises). */
int cfgms_deinterleave_host(cfgms_ctx* ctx, const int32_t* delayed, int32_t n, int32_t T, int32_t S,
                            int32_t* grid_out, void* cuda_stream);

/*
 * cfgms_deinterleave_host_static — cfgms_deinterleave_host for callers that must not allocate device memory
 * (same operation: grid[q][f][i] = delayed[q][f + i][i], 0 <= f < T - S + 1).
 *
 * Who needs it.  cfgms_create and cfgms_deinterleave_host call cudaMalloc (the latter whenever a batch is larger
 * than any it has seen).  That is not an option for every host program:
 *   - a serving engine of the kind the paper builds on hands almost all free HBM to its own cache pool at
 *     start-up; a cudaMalloc made later, when a request finishes and its codes have to be de-interleaved, can
 *     simply fail with out-of-memory although the work needs a few MiB;
 *   - cudaMalloc and cudaFree may synchronise the whole device, so a call made from the decode loop stalls every
 *     stream that is in flight, not only the caller's;
 *   - some deployments audit a fixed device-memory budget and forbid allocation after initialisation.
 * This entry point therefore takes NO context and calls no cudaMalloc, cudaFree, cudaMallocHost or any other
 * allocating routine, at set-up or later.  Its device staging (the uploaded delayed buffer and the grid before it
 * is copied back) lives in one array of CFGMS_STATIC_SCRATCH_BYTES that is part of the library image: every GPU
 * on which this process uses libcfgms.so holds those bytes from the moment the library's device code is loaded
 * there until the process exits, whether or not this function is ever called.
 *
 *   delayed  : HOST int32 [n][T][S]            grid_out : HOST int32 [n][T - S + 1][S]
 *   (pageable or pinned; only read / written during the call).  Requires T >= S >= 1, S <= 64, n <= 65535;
 *   n == 0 is a no-op.  Copies in on `cuda_stream`, runs the de-interleave kernel there, copies out and
 *   synchronises the stream before returning, like cfgms_deinterleave_host.
 *
 * Limit: round_up(n*T*S*4, 256) + n*(T-S+1)*S*4 <= CFGMS_STATIC_SCRATCH_BYTES (8 MiB: e.g. 64 requests of 1024
 * steps x 16 streams).  A larger request is refused with CFGMS_ERR_LIMIT before anything is copied or launched
 * and grid_out is left untouched; split the batch over several calls (requests are independent).
 *
 * First call on a device: the function looks up the array's device address (cudaGetSymbolAddress), checks that
 * the device is compute capability 10.x and raises the kernel's shared-memory limit.  This happens once per
 * device, on the calling thread, with that device current; make that first call during start-up, before any
 * stream capture is begun.  Later calls on the device do none of this.
 *
 * Sharing: all calls on one device use the SAME array and it keeps whatever the previous call left there.
 * Nothing in it has to start at zero — a call overwrites every word it later reads — so no clearing is done.
 * Two calls whose device work can overlap (different streams, or different threads) race on the array and
 * return garbage grids: order them yourself.  Calls from one thread are safe because each one returns only
 * after its stream has drained.
 * Errors: ARG, SHAPE, LIMIT, ARCH, CUDA (including "no device").
 */
#define CFGMS_STATIC_SCRATCH_BYTES (8u << 20)
int cfgms_deinterleave_host_static(const int32_t* delayed, int32_t n, int32_t T, int32_t S, int32_t* grid_out,
                                   void* cuda_stream);

/*
 * cfgms_last_device_error — reads the sticky device error word (one small D2H copy that
 * synchronises the device).  Returns CFGMS_OK or the latched status; *row_out (nullable)
 * receives the batch row it was raised for, or -1.  The word is cleared by the call.
 */
int cfgms_last_device_error(cfgms_ctx* ctx, int32_t* row_out);

typedef struct {
    int32_t S, d, V, max_rows, pad_token, num_sms;
    int32_t row_tile;              /* batch rows per accumulator tile of the last step          */
    int32_t row_blocks;            /* row tiles per vocabulary tile of the last step            */
    int32_t vocab_tiles;           /* ceil(S*V / 128)                                           */
    int32_t gemm_grid;             /* CTAs of the last head-GEMM launch                         */
    int32_t pipeline_stages;       /* TMA->MMA shared-memory ring depth of the last step        */
    int32_t launches_last_step;    /* kernels enqueued by the last cfgms_step                   */
    int64_t launches_total;        /* kernels enqueued since create                             */
    int64_t h2d_bytes_last_step;   /* cfgms_step_host only                                      */
    int64_t d2h_bytes_last_step;
    int32_t cta_pair;              /* 1 when the last head GEMM ran on CTA pairs (cta_group::2) */
    int32_t overlap;               /* 1 when the last finalize launch overlapped the head GEMM  */
    int32_t split_k;               /* 2 when the last head GEMM ran as split-K clusters of four CTAs, else 1 */
    int32_t reserved0;
} cfgms_info;
int cfgms_get_info(cfgms_ctx* ctx, cfgms_info* out);

/*
 * Profiling aid (bench.py's roofline figure).  While enabled, cfgms_step records CUDA events
 * on the launch stream before the head GEMM, between it and the finalize kernel, and after;
 * cfgms_profile_read waits for them and returns the summed device time of each kernel and the
 * number of recorded steps (at most 4096 between reads), then resets the ring.  Event records
 * perturb back-to-back launches slightly: time throughput with profiling off.
 */
int cfgms_profile_enable(cfgms_ctx* ctx, int on);
int cfgms_profile_read(cfgms_ctx* ctx, double* gemm_ms, double* finalize_ms, int64_t* steps);

/*
 * Evidence that the finalize kernel really runs beside the head GEMM (cfgms_info.overlap = 1):
 * *cells_waited = (request, stream) cells that reached their readiness check before the head
 * GEMM had finished their (stream, row block) group, i.e. while the GEMM was still running, since
 * the last call.  0 when the overlap is off.  One small D2H copy (synchronises the device);
 * resets the counter.
 */
int cfgms_overlap_stats(cfgms_ctx* ctx, int64_t* cells_waited);

const char* cfgms_strerror(int status);
/* Library build string: version, arch, compile flags. */
const char* cfgms_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CFGMS_H */
