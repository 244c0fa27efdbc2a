/*
 * cfgms_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the per-step audio decode head computes, written
 * from the paper (arxiv 2607.02119; citations are PAPER.md line numbers) and, where the paper
 * is silent, from the readings listed in DESIGN.md section 3 (ids C1..C20).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no source, header, table or helper with the CUDA path under
 * paper_2607_02119_b200/csrc/; the two only ever meet through the seeded inputs of workloads.py.
 *
 * Pins (tests/test_oracle_*.py): bf16 decode vs torch over all 65536 patterns; logits vs
 * torch fp64 matmul, linearity, hand-computed d=1 case; Eq. 1 identities at w=1, w=0 and
 * affinity in w; greedy vs numpy argmax; top-k by brute-force full sort; Philox4x32-10 vs the
 * CUDA toolkit's host-callable curand_Philox4x32_10; Gumbel-max frequencies vs softmax by a
 * chi-square bound; interleave/de-interleave identities and PAD counts.
 * Whole step: "parity unpinned" by the paper itself (it prints no worked numeric example);
 * every stage above is pinned separately.
 *
 * Steps (one call = one decode step over a batch of R rows):
 *   O1 decode bf16 bit patterns to double                                   (exact)
 *   O3 L[r][i][v] = sum_k W_i[v][k] * (h_r[k] + e_i[k]),  k ascending
 *   O4 paired:   M = w*L_cond + (1-w)*L_uncond   (Eq. 1 literally)
 *      unpaired: M = L
 *   O5 stream i active  <=>  i <= tau  and  tau < F + i  (0-based i)
 *   O6 greedy (top_k == 1 or temp == 0): argmax_v M, lowest v on ties
 *   O7 z = M / temp; thr = k-th largest z; keep = { v : z[v] >= thr }       (C8, C9, C10)
 *   O8 token = argmax_{v in keep} z[v] + g(v), g = -ln(-ln(1-p)),
 *      p = ((x >> 9) + 0.5) * 2^-23, x = word (v & 3) of
 *      Philox4x32-10(ctr = (v >> 2, tau, i, req_id), key = (seed_lo, seed_hi))   (C12)
 *   O9 tokens_out[cond] = tokens_out[uncond] = token
 *      delayed[c][tau mod T_cap][i] = token  (PAD when inactive)
 *   de-interleave: G[q][f][i] = D[q][f + i][i], F = T - S + 1
 * Widenings, each pinned in tests/test_oracle_widen.py:
 *   W1 oracle_emit_frame   streaming frame emission from the delay ring
 *      pin: emission over all steps == oracle_deinterleave of the full delayed matrix, for every
 *      ring depth >= S; hand-written 3-stream example
 *   W2 oracle_step_ex      static logit bias (vocabulary mask) + forced tokens
 *      pin: zero bias / no forcing == oracle_step bit-exactly; -inf mask == sampling on the
 *      reduced vocabulary (chi-square vs softmax over the unmasked tokens); forced cells verbatim
 *   W3 oracle_feedback     sum of the sampled tokens' stream embeddings
 *      pin: torch fp64 gather-sum; one stream == row copy; out-of-range ids contribute zero
 *   W4 oracle_advance_state  step counter, frame count set by end-of-audio, drained flag
 *      pin: a request driven by it to completion produces exactly interleave(grid of F frames):
 *      S(S-1)/2 PAD cells at each end, F + S - 1 steps, S - 1 PADs on the primary stream in the drain
 *   W6 oracle_phase_advance / oracle_step_phase  per-request phase state machine: text / transition /
 *      audio (+ drain) / done, vocabulary regions, CFG merge only in the audio phase, modality by argmax over
 *      the regions
 *      pin: hand-written traces of the transition function; an all-audio batch == oracle_step_ex bit-exactly;
 *      text-phase cells == a non-CFG run restricted to the text region (merge bypassed); region sampling ==
 *      -inf masking of the complement (W2's pinned mask); modality vs numpy argmax
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG 1
#define ORACLE_ERR_LAYOUT 3

/* flag bits written per cell */
#define ORC_INACTIVE 1   /* PAD cell, nothing sampled                                   */
#define ORC_GREEDY 2     /* took the explicit argmax branch O6                            */
#define ORC_CLOSE 4      /* best-minus-second perturbed score <= tol (north_star's rule)  */
#define ORC_BOUNDARY 8   /* outcome could change if z moved by < tol at the top-k edge    */
#define ORC_FORCED 16    /* token given by force_token, nothing sampled                   */

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- O1: bf16 <-> real ------------------------------------------------------------------- */
/* bf16 is the top 16 bits of an IEEE-754 binary32. */
static inline double bf16_to_double(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

void oracle_bf16_to_f64(const uint16_t* in, int64_t n, double* out) {
    for (int64_t j = 0; j < n; ++j) out[j] = bf16_to_double(in[j]);
}

/* fp32 -> bf16, round to nearest, ties to even (reading C18: config 1's fp32 hidden). */
void oracle_f32_to_bf16_rne(const float* in, int64_t n, uint16_t* out) {
    for (int64_t j = 0; j < n; ++j) {
        uint32_t u;
        memcpy(&u, &in[j], 4);
        if ((u & 0x7fffffffu) > 0x7f800000u) { /* NaN: keep it a quiet NaN */
            out[j] = (uint16_t)((u >> 16) | 0x0040u);
            continue;
        }
        uint32_t lower = u & 0xffffu;
        uint32_t upper = u >> 16;
        if (lower > 0x8000u || (lower == 0x8000u && (upper & 1u))) upper += 1u;
        out[j] = (uint16_t)upper;
    }
}

/* ---- Philox4x32-10 (Salmon et al., SC'11), restated from its definition ------------------ */
/* One round: two 32x32->64 multiplies by fixed odd constants, xor of the high halves with the
 * other two counter words and the key, and a word permutation.  The key is bumped by a Weyl
 * increment between rounds; ten rounds in all. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t MUL_A = 0xD2511F53u, MUL_B = 0xCD9E8D57u;
    const uint32_t WEYL_A = 0x9E3779B9u, WEYL_B = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += WEYL_A; k1 += WEYL_B; }
        uint64_t pa = (uint64_t)MUL_A * (uint64_t)c0;
        uint64_t pb = (uint64_t)MUL_B * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(pb >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)pb;
        uint32_t n2 = (uint32_t)(pa >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)pa;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* C12: 23 random bits -> p in (0,1), centred in its bin; exact in fp32 and fp64. */
double oracle_uniform(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* standard Gumbel from p: g = -ln(-ln(1-p)) */
double oracle_gumbel_from_uniform(double p) { return -log(-log1p(-p)); }

/* noise of token v for (seed, req_id, tau, stream) */
double oracle_gumbel(uint64_t seed, uint32_t req_id, int32_t tau, int32_t stream, int32_t v) {
    uint32_t ctr[4] = {(uint32_t)v >> 2, (uint32_t)tau, (uint32_t)stream, req_id};
    uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    uint32_t o[4];
    oracle_philox4x32_10(ctr, key, o);
    return oracle_gumbel_from_uniform(oracle_uniform(o[v & 3]));
}

/* ---- O3: head projection of one (row, stream) ------------------------------------------- */
/* out[v] = sum_{k=0}^{d-1} W_i[v][k] * (h_r[k] + e_i[k]) */
void oracle_logits_row(const uint16_t* heads, const uint16_t* embeds, const uint16_t* hidden,
                       int32_t S, int32_t d, int32_t V, int32_t row, int32_t stream, double* out) {
    (void)S;
    double* x = (double*)malloc(sizeof(double) * (size_t)d);
    const uint16_t* h = hidden + (size_t)row * d;
    const uint16_t* e = embeds + (size_t)stream * d;
    for (int32_t k = 0; k < d; ++k) x[k] = bf16_to_double(h[k]) + bf16_to_double(e[k]);
    const uint16_t* W = heads + (size_t)stream * V * d;
    for (int32_t v = 0; v < V; ++v) {
        const uint16_t* wr = W + (size_t)v * d;
        double acc = 0.0;
        for (int32_t k = 0; k < d; ++k) acc += bf16_to_double(wr[k]) * x[k];
        out[v] = acc;
    }
    free(x);
}

/* ---- O4: Eq. 1 ---------------------------------------------------------------------------- */
void oracle_cfg_merge(const double* l_cond, const double* l_uncond, double w, int32_t V, double* out) {
    for (int32_t v = 0; v < V; ++v) out[v] = w * l_cond[v] + (1.0 - w) * l_uncond[v];
}

/* ---- O6-O8: sampling of one cell from its merged logits ---------------------------------- */
static int cmp_desc(const void* a, const void* b) {
    double x = *(const double*)a, y = *(const double*)b;
    return (x < y) - (x > y);
}

/* Returns the token. margin = best - second best perturbed score inside keep (+inf if alone).
 * flags: ORC_GREEDY / ORC_CLOSE / ORC_BOUNDARY.  thr_out (nullable) = top-k threshold on z.
 * M holds the V logits of tokens v_off .. v_off + V - 1 (a vocabulary REGION, widening W6; v_off = 0
 * for a whole sub-vocabulary): the returned token is region-local, the noise of entry v is keyed by
 * its global token id v_off + v. */
static int32_t sample_cell_region(const double* M, int32_t V, int32_t v_off, float temp, int32_t top_k, uint64_t seed,
                                  uint32_t req_id, int32_t tau, int32_t stream, double tol,
                                  double* margin_out, int32_t* flags_out, double* thr_out) {
    int32_t flags = 0;
    double margin = INFINITY;
    int32_t tok = 0;
    if (top_k == 1 || temp == 0.0f) { /* O6 */
        flags |= ORC_GREEDY;
        for (int32_t v = 1; v < V; ++v) if (M[v] > M[tok]) tok = v;
        for (int32_t v = 0; v < V; ++v) if (v != tok && M[tok] - M[v] < margin) margin = M[tok] - M[v];
        if (thr_out) *thr_out = M[tok];
    } else {
        double* z = (double*)malloc(sizeof(double) * (size_t)V * 3);
        double* sorted = z + V;
        double* s = z + 2 * (size_t)V;
        double t = (double)temp;
        for (int32_t v = 0; v < V; ++v) z[v] = M[v] / t;                    /* O7 */
        int32_t k = (top_k <= 0 || top_k >= V) ? V : top_k;
        memcpy(sorted, z, sizeof(double) * (size_t)V);
        qsort(sorted, (size_t)V, sizeof(double), cmp_desc);
        double thr = sorted[k - 1];
        if (thr_out) *thr_out = thr;
        int first = 1;
        for (int32_t v = 0; v < V; ++v) {                                    /* O8 */
            if (z[v] >= thr) {
                s[v] = z[v] + oracle_gumbel(seed, req_id, tau, stream, v_off + v);
                if (first || s[v] > s[tok]) { tok = v; first = 0; }
            }
        }
        for (int32_t v = 0; v < V; ++v)
            if (v != tok && z[v] >= thr && s[tok] - s[v] < margin) margin = s[tok] - s[v];
        /* top-k edge: would a perturbation of z by < tol change who may compete? */
        if (z[tok] < thr + tol && k < V) flags |= ORC_BOUNDARY;
        for (int32_t v = 0; v < V; ++v) {
            if (z[v] < thr && z[v] >= thr - tol) {
                double sv = z[v] + oracle_gumbel(seed, req_id, tau, stream, v_off + v);
                if (sv >= s[tok] - tol) flags |= ORC_BOUNDARY;
            }
        }
        free(z);
    }
    if (margin <= tol) flags |= ORC_CLOSE;
    if (margin_out) *margin_out = margin;
    if (flags_out) *flags_out = flags;
    return tok;
}

int32_t oracle_sample_cell(const double* M, int32_t V, float temp, int32_t top_k, uint64_t seed,
                           uint32_t req_id, int32_t tau, int32_t stream, double tol,
                           double* margin_out, int32_t* flags_out, double* thr_out) {
    return sample_cell_region(M, V, 0, temp, top_k, seed, req_id, tau, stream, tol, margin_out, flags_out, thr_out);
}

/* ---- O2: batch layout contract ------------------------------------------------------------ */
/* cond row even, pair_map[c] = c+1, pair_map[c+1] = c; unpaired rows carry -1. */
int oracle_check_pair_map(const int32_t* pair_map, int32_t R) {
    for (int32_t r = 0; r < R; ++r) {
        int32_t p = pair_map[r];
        if (p == -1) continue;
        if (p < 0 || p >= R) return ORACLE_ERR_LAYOUT;
        if (pair_map[p] != r) return ORACLE_ERR_LAYOUT;
        if ((r % 2 == 0 && p != r + 1) || (r % 2 == 1 && p != r - 1)) return ORACLE_ERR_LAYOUT;
    }
    return ORACLE_OK;
}

/* ---- one decode step --------------------------------------------------------------------- */
/* cells: nullable int32 [n_cells][2] = (request-owning row c, stream i); NULL => every
 * request-owning row x every stream, in row-major order, and n_cells is ignored.
 * Per evaluated cell j (in list order): tok_out[j], margin_out[j], flags_out[j], and if
 * merged_out != NULL merged_out[j][V] (pre-temperature merged logits, zeros for PAD cells).
 * tokens_out [R][S] and delayed [R][T_cap][S] (both nullable) receive O9's writes for the
 * evaluated cells only; other entries are left untouched. */
/* Widening W2 (the hooks through which the phase state machine of
 * PAPER.md:70-76 acts on the audio head):
 *   logit_bias  nullable double [S][V]: merged logits become M + bias[i][v] BEFORE the
 *               temperature ("dynamic vocabulary masking": -inf removes a token);
 *   force_token nullable int32 [R][S], read at the request-owning row: a value >= 0 is emitted
 *               as the cell's token without sampling (a deterministic bridging token of the
 *               transition phase, or the padding of a text-phase row); < 0 = sample normally.
 *               It is only consulted for ACTIVE cells: the delay pattern's PAD wins. */
int oracle_step_ex(const uint16_t* heads, const uint16_t* embeds, const uint16_t* hidden,
                   int32_t R, int32_t S, int32_t d, int32_t V,
                   const int32_t* pair_map, const float* w, const float* temp, const int32_t* top_k,
                   uint64_t seed, const int32_t* step, const uint32_t* req_id, const int32_t* n_frames,
                   int32_t pad_token, double tol,
                   const int32_t* cells, int64_t n_cells,
                   int32_t* tok_out, double* margin_out, int32_t* flags_out, double* merged_out,
                   int32_t* tokens_out, int32_t* delayed, int32_t T_cap,
                   const double* logit_bias, const int32_t* force_token) {
    if (R <= 0 || S <= 0 || d <= 0 || V <= 0) return ORACLE_ERR_ARG;
    int rc = oracle_check_pair_map(pair_map, R);
    if (rc != ORACLE_OK) return rc;

    int32_t* all_cells = NULL;
    if (cells == NULL) {
        int64_t n = 0;
        for (int32_t r = 0; r < R; ++r) if (pair_map[r] < 0 || r % 2 == 0) n += S;
        all_cells = (int32_t*)malloc(sizeof(int32_t) * 2 * (size_t)n);
        int64_t j = 0;
        for (int32_t r = 0; r < R; ++r)
            if (pair_map[r] < 0 || r % 2 == 0)
                for (int32_t i = 0; i < S; ++i) { all_cells[2 * j] = r; all_cells[2 * j + 1] = i; ++j; }
        cells = all_cells;
        n_cells = n;
    }
    for (int64_t j = 0; j < n_cells; ++j) {
        int32_t c = cells[2 * j], i = cells[2 * j + 1];
        if (c < 0 || c >= R || i < 0 || i >= S || (pair_map[c] >= 0 && c % 2 == 1)) {
            free(all_cells);
            return ORACLE_ERR_ARG;
        }
    }

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n_cells; ++j) {
        int32_t c = cells[2 * j], i = cells[2 * j + 1];
        int32_t u = pair_map[c];
        int32_t tau = step[c];
        uint32_t rid = req_id ? req_id[c] : (uint32_t)c;
        int32_t tok, flags = 0;
        double margin = INFINITY;
        int active = (i <= tau) && (n_frames == NULL || tau - i < n_frames[c]);      /* O5: tau < F + i, written without the sum so that F = INT32_MAX ("no frame count yet", C27) cannot overflow */
        if (!active) {
            tok = pad_token;
            flags = ORC_INACTIVE;
            if (merged_out) memset(merged_out + (size_t)j * V, 0, sizeof(double) * (size_t)V);
        } else if (force_token && force_token[(size_t)c * S + i] >= 0) {
            tok = force_token[(size_t)c * S + i];
            flags = ORC_FORCED;
            if (merged_out) memset(merged_out + (size_t)j * V, 0, sizeof(double) * (size_t)V);
        } else {
            double* Lc = (double*)malloc(sizeof(double) * (size_t)V * 3);
            double* Lu = Lc + V;
            double* M = Lc + 2 * (size_t)V;
            oracle_logits_row(heads, embeds, hidden, S, d, V, c, i, Lc);             /* O3 */
            if (u >= 0) {
                oracle_logits_row(heads, embeds, hidden, S, d, V, u, i, Lu);
                oracle_cfg_merge(Lc, Lu, (double)w[c], V, M);                        /* O4 */
            } else {
                memcpy(M, Lc, sizeof(double) * (size_t)V);
            }
            if (logit_bias)
                for (int32_t v = 0; v < V; ++v) M[v] += logit_bias[(size_t)i * V + v];
            tok = oracle_sample_cell(M, V, temp[c], top_k[c], seed, rid, tau, i, tol,
                                     &margin, &flags, NULL);                         /* O6-O8 */
            if (merged_out) memcpy(merged_out + (size_t)j * V, M, sizeof(double) * (size_t)V);
            free(Lc);
        }
        if (tok_out) tok_out[j] = tok;
        if (margin_out) margin_out[j] = margin;
        if (flags_out) flags_out[j] = flags;
        if (tokens_out) {                                                            /* O9 */
            tokens_out[(size_t)c * S + i] = tok;
            if (u >= 0) tokens_out[(size_t)u * S + i] = tok;
        }
        if (delayed && T_cap > 0) {
            int32_t slot = ((tau % T_cap) + T_cap) % T_cap;
            delayed[((size_t)c * T_cap + slot) * S + i] = tok;
        }
    }
    free(all_cells);
    return ORACLE_OK;
}

int oracle_step(const uint16_t* heads, const uint16_t* embeds, const uint16_t* hidden,
                int32_t R, int32_t S, int32_t d, int32_t V,
                const int32_t* pair_map, const float* w, const float* temp, const int32_t* top_k,
                uint64_t seed, const int32_t* step, const uint32_t* req_id, const int32_t* n_frames,
                int32_t pad_token, double tol,
                const int32_t* cells, int64_t n_cells,
                int32_t* tok_out, double* margin_out, int32_t* flags_out, double* merged_out,
                int32_t* tokens_out, int32_t* delayed, int32_t T_cap) {
    return oracle_step_ex(heads, embeds, hidden, R, S, d, V, pair_map, w, temp, top_k, seed, step, req_id,
                          n_frames, pad_token, tol, cells, n_cells, tok_out, margin_out, flags_out,
                          merged_out, tokens_out, delayed, T_cap, NULL, NULL);
}

/* ---- delay pattern ------------------------------------------------------------------------ */
/* grid[q][f][i] = delayed[q][f + i][i], 0 <= f < F = T - S + 1 */
int oracle_deinterleave(const int32_t* delayed, int32_t n, int32_t T, int32_t S, int32_t* grid) {
    if (n < 0 || S <= 0 || T < S) return ORACLE_ERR_ARG;
    int32_t F = T - S + 1;
    for (int32_t q = 0; q < n; ++q)
        for (int32_t f = 0; f < F; ++f)
            for (int32_t i = 0; i < S; ++i)
                grid[((size_t)q * F + f) * S + i] = delayed[((size_t)q * T + (f + i)) * S + i];
    return ORACLE_OK;
}

/* delayed[q][t][i] = (0 <= t - i < F) ? grid[q][t - i][i] : PAD,  T = F + S - 1 */
int oracle_interleave(const int32_t* grid, int32_t n, int32_t F, int32_t S, int32_t pad, int32_t* delayed) {
    if (n < 0 || S <= 0 || F <= 0) return ORACLE_ERR_ARG;
    int32_t T = F + S - 1;
    for (int32_t q = 0; q < n; ++q)
        for (int32_t t = 0; t < T; ++t)
            for (int32_t i = 0; i < S; ++i) {
                int32_t f = t - i;
                delayed[((size_t)q * T + t) * S + i] =
                    (f >= 0 && f < F) ? grid[((size_t)q * F + f) * S + i] : pad;
            }
    return ORACLE_OK;
}

/* Widening W1 — streaming finished-frame emission ("fusing waveform synthesis
 * directly into the serving path", Fig. 2 left).  After step tau of a
 * request whose delayed tokens live in a ring of depth T_cap >= S (ring[t mod T_cap][i] = token
 * of stream i sampled at step t), frame f = tau - S + 1 is complete iff 0 <= f < F:
 *     frame[i] = ring[(f + i) mod T_cap][i]        (= D[f + i][i], the de-interleave rule)
 * Returns f, or -1 when no frame completes at this step (frame[] is then filled with pad). */
int32_t oracle_emit_frame(const int32_t* ring, int32_t T_cap, int32_t S, int32_t tau, int32_t F,
                          int32_t pad, int32_t* frame) {
    int32_t f = tau - S + 1;
    if (f < 0 || (F >= 0 && f >= F) || T_cap < S) {
        for (int32_t i = 0; i < S; ++i) frame[i] = pad;
        return -1;
    }
    for (int32_t i = 0; i < S; ++i) frame[i] = ring[(size_t)((f + i) % T_cap) * S + i];
    return f;
}

/* Widening W3 — autoregressive feedback aggregation ("the input representation at
 * each step aggregates the embeddings of these previously generated tokens"; reading C25: the
 * aggregate is the SUM over the S streams of the stream's own embedding row of its token).
 *     x[r][k] = sum_{i=0}^{S-1} Emb_i[tokens[r][i]][k]        i ascending, fp64
 * emb: bf16 [S][V_e][d]; a token id outside [0, V_e) contributes nothing. */
void oracle_feedback(const int32_t* tokens, const uint16_t* emb, int32_t R, int32_t S, int32_t V_e, int32_t d,
                     double* x) {
    for (int32_t r = 0; r < R; ++r)
        for (int32_t k = 0; k < d; ++k) {
            double acc = 0.0;
            for (int32_t i = 0; i < S; ++i) {
                int32_t t = tokens[(size_t)r * S + i];
                if (t >= 0 && t < V_e) acc += bf16_to_double(emb[((size_t)i * V_e + t) * d + k]);
            }
            x[(size_t)r * d + k] = acc;
        }
}

/* Widening W4 — device-resident request state with automatic drain ("terminating the
 * audio phase initiates a drain sub-phase that emits S-1 padding tokens to flush the delay buffer,
 * guaranteeing a complete S x T codebook matrix"; reading C27: the audio phase of a request ends
 * when its PRIMARY stream (stream 0) emits the end-of-audio token at step tau; the frames completed
 * so far, F = tau, become the request's frame count, stream 0 pads from then on and stream i keeps
 * sampling its delayed tokens for i more steps).  `unset` marks "no frame count yet".
 *   in : tau, F (or unset), tok0 = the token stream 0 emitted at this step, eos (< 0: none)
 *   out: *tau_next = tau + 1;  *F_next = F, or tau if F was unset and tok0 == eos;
 *        returns 1 iff the request is fully drained after this step: tau + 1 >= F_next + S - 1. */
int32_t oracle_advance_state(int32_t tau, int32_t F, int32_t tok0, int32_t eos, int32_t S, int32_t unset,
                             int32_t* tau_next, int32_t* F_next) {
    int32_t Fn = F;
    if (F == unset && eos >= 0 && tok0 == eos) Fn = tau;
    *tau_next = tau + 1;
    *F_next = Fn;
    return (Fn != unset && tau + 1 >= Fn + S - 1) ? 1 : 0;
}

/* ---- test helper: empirical token frequencies of O6-O8 on fixed merged logits ------------- */
/* counts[v] += 1 for each of the n_req * n_tau draws obtained by sweeping (req_id, tau). */
void oracle_sample_sweep(const double* M, int32_t V, float temp, int32_t top_k, uint64_t seed,
                         int32_t n_req, int32_t n_tau, int32_t stream, int64_t* counts) {
    for (int32_t q = 0; q < n_req; ++q)
        for (int32_t tau = 0; tau < n_tau; ++tau) {
            int32_t tok = oracle_sample_cell(M, V, temp, top_k, seed, (uint32_t)q, tau, stream, 0.0,
                                             NULL, NULL, NULL);
            counts[tok] += 1;
        }
}


/* ---- Widening W6 — per-request phase state machine (readings C28-C32 of DESIGN.md) ----
 * "a per-request phase state machine enforced via dynamic vocabulary masking ... a text phase restricted
 * to text tokens, a transition phase injecting deterministic bridging tokens to condition audio
 * generation, and an audio phase activating all S streams ... terminating the audio phase initiates a
 * drain sub-phase that emits S-1 padding tokens ... dynamically inferring the active modality directly
 * from the model's unmasked output distribution (i.e., the argmax over the disjoint vocabulary regions)"
 * and "this CFG merge operates only during the audio phase; it bypasses modality-switching
 * tokens".
 *
 * C28 the PRIMARY stream (stream 0) is the one that carries text: its V logits cover the disjoint regions
 *     [0, V_text) = text tokens and [V_text, V) = its audio codes (and the end-of-audio id); streams >= 1
 *     are audio only.  "Dynamic vocabulary masking" = the phase selects the region a cell may sample from.
 * C29 TEXT: only stream 0 samples, from the text region, from the CONDITIONAL row's logits alone (no merge);
 *     streams >= 1 emit PAD.  The modality the model asks for is the region of argmax_v of the UNMASKED
 *     logits of stream 0 (lowest v on ties); when it is the audio region, the request leaves the text phase
 *     AFTER this step (the step's token is still the text token it sampled).
 * C30 TRANSITION: stream 0 emits the deterministic bridging tokens bridge[0..n_bridge-1], one per step,
 *     streams >= 1 emit PAD, nothing is sampled; then the audio phase starts with audio-local step 0.
 * C31 AUDIO: rows a1-a4 of the hot path with the audio-local step tau_a (delay pattern, frame count, ring
 *     slot), stream 0 restricted to its audio region; the end-of-audio token on stream 0 fixes the frame count
 *     (W4) and the drain runs S-1 more steps; then DONE (every stream PAD, state frozen).
 * C32 the noise is keyed by the request's GLOBAL step (monotone over all phases), never by the phase-local
 *     position, so no two steps of a request share noise.
 *
 * One transition.  `pos` = bridging tokens emitted so far (TRANSITION) or the audio-local step tau_a (AUDIO).
 * tok0 = stream 0's token of this step; modality_audio = C29's inference (only read in TEXT).
 * Returns 1 iff the request is DONE after this step. */
#define ORC_PHASE_TEXT 0
#define ORC_PHASE_TRANSITION 1
#define ORC_PHASE_AUDIO 2
#define ORC_PHASE_DONE 3

int32_t oracle_phase_advance(int32_t phase, int32_t pos, int32_t F, int32_t tok0, int32_t modality_audio,
                             int32_t n_bridge, int32_t eos, int32_t S, int32_t unset,
                             int32_t* phase_next, int32_t* pos_next, int32_t* F_next) {
    int32_t pn = phase, qn = pos, Fn = F;
    if (phase == ORC_PHASE_TEXT) {
        qn = 0;
        if (modality_audio) pn = n_bridge > 0 ? ORC_PHASE_TRANSITION : ORC_PHASE_AUDIO;
    } else if (phase == ORC_PHASE_TRANSITION) {
        if (pos + 1 >= n_bridge) { pn = ORC_PHASE_AUDIO; qn = 0; }
        else qn = pos + 1;
    } else if (phase == ORC_PHASE_AUDIO) {
        int32_t tn;
        int32_t drained = oracle_advance_state(pos, F, tok0, eos, S, unset, &tn, &Fn);   /* W4 with tau = tau_a */
        qn = tn;
        if (drained) pn = ORC_PHASE_DONE;
    }
    *phase_next = pn; *pos_next = qn; *F_next = Fn;
    return pn == ORC_PHASE_DONE ? 1 : 0;
}

/* One decode step of a batch whose requests sit in different phases.  Arguments as oracle_step_ex, plus
 *   phase, pos    int32 [R], read at the request-owning row (C29-C31)
 *   gstep         int32 [R] the request's global step: keys the noise (C32)
 *   V_text        size of stream 0's text region (C28), 0 <= V_text <= V
 *   bridge        int32 [n_bridge] bridging tokens (C30)
 * n_frames [R] (nullable = unset) is relative to the audio-local step.  Per evaluated cell j: tok_out,
 * margin_out, flags_out, merged_out (the logits the cell sampled from BEFORE the region restriction: cond-only
 * in TEXT, merged in AUDIO; zeros where nothing was sampled).  Per evaluated cell of stream 0 additionally
 * modality_out[j] = 1 when C29's argmax lies in the audio region (0 elsewhere).  tokens_out / delayed as in
 * oracle_step_ex, except that only AUDIO-phase cells write the delayed buffer, at slot tau_a mod T_cap. */
int oracle_step_phase(const uint16_t* heads, const uint16_t* embeds, const uint16_t* hidden,
                      int32_t R, int32_t S, int32_t d, int32_t V,
                      const int32_t* pair_map, const float* w, const float* temp, const int32_t* top_k,
                      uint64_t seed, const int32_t* gstep, const uint32_t* req_id, const int32_t* n_frames,
                      int32_t pad_token, double tol,
                      const int32_t* cells, int64_t n_cells,
                      int32_t* tok_out, double* margin_out, int32_t* flags_out, double* merged_out,
                      int32_t* tokens_out, int32_t* delayed, int32_t T_cap,
                      const double* logit_bias,
                      const int32_t* phase, const int32_t* pos, int32_t V_text,
                      const int32_t* bridge, int32_t n_bridge, int32_t* modality_out) {
    if (R <= 0 || S <= 0 || d <= 0 || V <= 0 || !cells || !phase || !pos || V_text < 0 || V_text > V) return ORACLE_ERR_ARG;
    int rc = oracle_check_pair_map(pair_map, R);
    if (rc != ORACLE_OK) return rc;
    for (int64_t j = 0; j < n_cells; ++j) {
        int32_t c = cells[2 * j], i = cells[2 * j + 1];
        if (c < 0 || c >= R || i < 0 || i >= S || (pair_map[c] >= 0 && c % 2 == 1)) return ORACLE_ERR_ARG;
        if (phase[c] == ORC_PHASE_TRANSITION && (pos[c] < 0 || pos[c] >= n_bridge)) return ORACLE_ERR_ARG;
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n_cells; ++j) {
        int32_t c = cells[2 * j], i = cells[2 * j + 1];
        int32_t u = pair_map[c];
        int32_t ph = phase[c], q = pos[c];
        uint32_t rid = req_id ? req_id[c] : (uint32_t)c;
        int32_t tok = pad_token, flags = ORC_INACTIVE, modality = 0;
        double margin = INFINITY;
        int sample = 0, merge = 0;
        int32_t lo = 0, hi = V;
        if (ph == ORC_PHASE_TEXT) {                                   /* C29 */
            if (i == 0) { sample = 1; merge = 0; lo = 0; hi = V_text; }
        } else if (ph == ORC_PHASE_TRANSITION) {                      /* C30 */
            if (i == 0) { tok = bridge[q]; flags = ORC_FORCED; }
        } else if (ph == ORC_PHASE_AUDIO) {                           /* C31: O5 with tau_a */
            int active = (i <= q) && (n_frames == NULL || q - i < n_frames[c]);
            if (active) { sample = 1; merge = 1; lo = i == 0 ? V_text : 0; hi = V; }
        }
        if (merged_out) memset(merged_out + (size_t)j * V, 0, sizeof(double) * (size_t)V);
        if (sample) {
            double* Lc = (double*)malloc(sizeof(double) * (size_t)V * 3);
            double* Lu = Lc + V;
            double* M = Lc + 2 * (size_t)V;
            oracle_logits_row(heads, embeds, hidden, S, d, V, c, i, Lc);                          /* O3 */
            if (merge && u >= 0) {
                oracle_logits_row(heads, embeds, hidden, S, d, V, u, i, Lu);
                oracle_cfg_merge(Lc, Lu, (double)w[c], V, M);                                     /* O4, audio phase only */
            } else {
                memcpy(M, Lc, sizeof(double) * (size_t)V);
            }
            if (logit_bias)
                for (int32_t v = 0; v < V; ++v) M[v] += logit_bias[(size_t)i * V + v];
            if (ph == ORC_PHASE_TEXT) {                                                           /* C29: unmasked argmax */
                int32_t am = 0;
                for (int32_t v = 1; v < V; ++v) if (M[v] > M[am]) am = v;
                modality = am >= V_text ? 1 : 0;
            }
            flags = 0;
            if (hi > lo) {
                tok = lo + sample_cell_region(M + lo, hi - lo, lo, temp[c], top_k[c], seed, rid, gstep[c], i, tol,
                                              &margin, &flags, NULL);                              /* O6-O8 on the region */
            } else {
                tok = pad_token; flags = ORC_INACTIVE;      /* empty region: nothing to sample */
            }
            if (merged_out) memcpy(merged_out + (size_t)j * V, M, sizeof(double) * (size_t)V);
            free(Lc);
        }
        if (tok_out) tok_out[j] = tok;
        if (margin_out) margin_out[j] = margin;
        if (flags_out) flags_out[j] = flags;
        if (modality_out) modality_out[j] = modality;
        if (tokens_out) {                                                                         /* O9 */
            tokens_out[(size_t)c * S + i] = tok;
            if (u >= 0) tokens_out[(size_t)u * S + i] = tok;
        }
        if (delayed && T_cap > 0 && ph == ORC_PHASE_AUDIO) {
            int32_t slot = ((q % T_cap) + T_cap) % T_cap;
            delayed[((size_t)c * T_cap + slot) * S + i] = tok;
        }
    }
    return ORACLE_OK;
}
