"""Pins for the oracle's widening functions:
W1 streaming frame emission, W2 static logit bias + forced tokens, W3 feedback aggregation,
W4 request-state advance with automatic drain.  CPU only; every check compares the oracle with something other than itself."""
import numpy as np
import torch
from scipy import stats

import oracle
import workloads


# ------------------------------------------------------------------ W1: frame emission
def _drive_ring(grid, pad, T_cap):
    """Play a [F][S] grid through the delay pattern step by step into a ring of depth T_cap,
    emitting frames as they complete.  The delayed matrix comes from the interleave rule written
    out here (not from oracle.interleave)."""
    F, S = grid.shape
    T = F + S - 1
    ring = np.full((T_cap, S), -7, dtype=np.int32)
    frames = {}
    for tau in range(T):
        for i in range(S):
            f = tau - i
            ring[tau % T_cap, i] = grid[f, i] if 0 <= f < F else pad
        fi, fr = oracle.emit_frame(ring, tau, F, pad)
        if fi >= 0:
            assert fi not in frames
            frames[fi] = fr.copy()
        else:
            assert np.all(fr == pad)
    return frames


def test_emit_frame_hand_example():
    # S = 3, ring depth 3.  After step tau = 4 the ring holds steps 2, 3, 4 and frame 2 is
    # (stream 0 @ step 2, stream 1 @ step 3, stream 2 @ step 4)  -- PAPER.md:56 "i-th stream offset by i steps"
    ring = np.zeros((3, 3), dtype=np.int32)
    ring[2 % 3] = [20, 21, 22]    # step 2
    ring[3 % 3] = [30, 31, 32]    # step 3
    ring[4 % 3] = [40, 41, 42]    # step 4
    f, fr = oracle.emit_frame(ring, 4, 10, 99)
    assert f == 2 and fr.tolist() == [20, 31, 42]
    # before the first frame completes, and after the last one
    assert oracle.emit_frame(ring, 1, 10, 99)[0] == -1
    f, fr = oracle.emit_frame(ring, 12, 10, 99)      # f = 10 >= F
    assert f == -1 and fr.tolist() == [99, 99, 99]
    assert oracle.emit_frame(ring, 11, 10, 99)[0] == 9   # last frame


def test_emit_frame_over_all_steps_is_the_deinterleave():
    rng = np.random.default_rng(5)
    for S in (1, 2, 3, 4, 8, 16):
        for F in (1, 2, 5, 23):
            grid = rng.integers(0, 1000, size=(F, S), dtype=np.int32)
            for T_cap in (S, S + 1, 2 * S + 3, F + S - 1):
                frames = _drive_ring(grid, pad=1000, T_cap=T_cap)
                assert sorted(frames) == list(range(F))
                got = np.stack([frames[f] for f in range(F)])
                assert np.array_equal(got, grid)
                # and it equals the oracle's bulk de-interleave of the full delayed matrix
                dl = oracle.interleave(grid[None], 1000)
                assert np.array_equal(oracle.deinterleave(dl)[0], got)


def test_emit_frame_needs_ring_depth_S():
    ring = np.zeros((2, 3), dtype=np.int32)
    assert oracle.emit_frame(ring, 5, 10, 9)[0] == -1     # T_cap < S: nothing can be complete


# ------------------------------------------------------------------ W3: feedback aggregation
def test_feedback_vs_torch_gather_sum():
    g = torch.Generator().manual_seed(3)
    S, V_e, d, R = 5, 37, 48, 9
    emb = torch.randn(S, V_e, d, generator=g).to(torch.bfloat16)
    tok = torch.randint(0, V_e, (R, S), generator=g, dtype=torch.int32)
    want = torch.zeros(R, d, dtype=torch.float64)
    for i in range(S):
        want += emb[i].to(torch.float64)[tok[:, i].long()]
    got = oracle.feedback(tok.numpy(), emb)
    assert np.allclose(got, want.numpy(), rtol=0, atol=1e-12)


def test_feedback_single_stream_is_a_row_copy_and_out_of_range_is_zero():
    g = torch.Generator().manual_seed(4)
    S, V_e, d = 3, 11, 16
    emb = torch.randn(S, V_e, d, generator=g).to(torch.bfloat16)
    e64 = emb.to(torch.float64).numpy()
    tok = np.array([[4, -1, V_e], [-5, 2, 99], [-1, -1, -1], [0, 0, 0]], dtype=np.int32)
    x = oracle.feedback(tok, emb)
    assert np.array_equal(x[0], e64[0, 4])          # only stream 0 in range: exact copy
    assert np.array_equal(x[1], e64[1, 2])
    assert np.all(x[2] == 0.0)
    assert np.allclose(x[3], e64[0, 0] + e64[1, 0] + e64[2, 0], atol=1e-15)
    # stream i uses ITS OWN table: swapping two streams' tokens changes the result
    a = oracle.feedback(np.array([[1, 2, 3]], dtype=np.int32), emb)
    b = oracle.feedback(np.array([[2, 1, 3]], dtype=np.int32), emb)
    assert not np.allclose(a, b)
    assert np.allclose(a[0], e64[0, 1] + e64[1, 2] + e64[2, 3], atol=1e-15)


# ------------------------------------------------------------------ W2: logit bias + forced tokens
def _tiny():
    wl = workloads.make_config(1)
    t = 6     # every stream active (S = 4)
    return wl, t


def _run(wl, t, **kw):
    return oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                       wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, want_merged=True,
                       hidden_is_f32=wl.hidden_f32, **kw)


def test_zero_bias_and_no_forcing_change_nothing():
    wl, t = _tiny()
    base = _run(wl, t)
    ext = _run(wl, t, logit_bias=np.zeros((wl.S, wl.V)), force_token=np.full((wl.R, wl.S), -1, dtype=np.int32))
    assert np.array_equal(base.tok, ext.tok) and np.array_equal(base.merged, ext.merged)
    assert np.array_equal(base.flags, ext.flags) and np.array_equal(base.margin, ext.margin)


def test_bias_is_added_to_the_merged_logits_before_temperature():
    wl, t = _tiny()
    rng = np.random.default_rng(2)
    bias = rng.normal(size=(wl.S, wl.V))
    base, ext = _run(wl, t), _run(wl, t, logit_bias=bias)
    for j, (c, i) in enumerate(base.cells):
        assert np.array_equal(ext.merged[j], base.merged[j] + bias[i])     # same fp64 add, stream's own row
    # a huge bonus on one token makes it the sampled token of that stream for every request
    bonus = np.zeros((wl.S, wl.V))
    bonus[2, 17] = 1e4
    forced = _run(wl, t, logit_bias=bonus)
    for j, (c, i) in enumerate(forced.cells):
        assert (forced.tok[j] == 17) == (i == 2) or base.tok[j] == 17


def test_minus_inf_mask_equals_sampling_on_the_reduced_vocabulary():
    # Gumbel-max over M + mask must follow softmax over the UNMASKED tokens only (textbook
    # identity); checked by a chi-square bound on 2^16 draws, and no masked token may ever appear.
    V = 16
    rng = np.random.default_rng(9)
    M = rng.normal(scale=1.5, size=V)
    mask = np.zeros(V)
    masked = [1, 4, 5, 11, 15]
    mask[masked] = -np.inf
    counts = oracle.sample_sweep(M + mask, temp=0.7, top_k=0, seed=77, n_req=256, n_tau=256)
    assert counts[masked].sum() == 0
    keep = [v for v in range(V) if v not in masked]
    p = np.exp(M[keep] / 0.7)
    p /= p.sum()
    n = counts.sum()
    chi2 = float((((counts[keep] - n * p) ** 2) / (n * p)).sum())
    assert chi2 <= stats.chi2.ppf(1 - 1e-6, len(keep) - 1)
    # with top-k: the k largest UNMASKED tokens compete
    counts = oracle.sample_sweep(M + mask, temp=0.7, top_k=4, seed=78, n_req=64, n_tau=64)
    top4 = sorted(keep, key=lambda v: -M[v])[:4]
    assert counts.sum() == counts[top4].sum() and all(counts[v] > 0 for v in top4)


def test_forced_tokens_are_emitted_verbatim_and_only_in_active_cells():
    wl, _ = _tiny()
    ft = np.full((wl.R, wl.S), -1, dtype=np.int32)
    ft[0, 1] = 200           # cond row of pair 0, stream 1: bridging token
    ft[0, 3] = 201           # stream 3 is not active yet at step 2: the delay pattern's PAD wins
    ft[1, 2] = 123           # companion row: ignored (parameters are read at the cond row)
    tokens = np.full((wl.R, wl.S), -1, dtype=np.int32)
    t = 2
    base = _run(wl, t)
    ext = _run(wl, t, force_token=ft, tokens_out=tokens)
    for j, (c, i) in enumerate(ext.cells):
        if (c, i) == (0, 1):
            assert ext.tok[j] == 200 and ext.flags[j] & oracle.FLAG_FORCED
        elif (c, i) == (0, 3):
            assert ext.tok[j] == wl.pad_token and ext.flags[j] & oracle.FLAG_INACTIVE
        else:
            assert ext.tok[j] == base.tok[j] and ext.flags[j] == base.flags[j]
    assert tokens[0, 1] == 200 and tokens[1, 1] == 200      # synchronised to the companion


# ------------------------------------------------------------------ W4: device-resident state, automatic drain
def test_state_machine_drives_a_request_to_a_complete_codebook_matrix():
    """ending the audio phase starts a drain that emits S-1 paddings on the primary stream and
    guarantees a complete matrix.  Drive one request with oracle.advance_state only (tokens are arbitrary
    symbols here; the end-of-audio symbol appears on stream 0 at a chosen step) and check the result
    against the interleave rule written out independently: F frames, F + S - 1 steps, PAD exactly
    where t - i is outside [0, F)."""
    EOS, PAD = 777, 1000
    for S in (1, 2, 4, 9):
        for F_true in (0, 1, 3, 11):
            tau, F, rows, done, steps = 0, oracle.F_UNSET, [], False, 0
            while not done:
                row = []
                for i in range(S):
                    active = i <= tau and (tau - i < F)          # activity rule O5 with the CURRENT frame count
                    tok = PAD if not active else (EOS if (i == 0 and tau == F_true) else 10 * tau + i)
                    row.append(tok)
                rows.append(row)
                tau, F, done = oracle.advance_state(tau, F, row[0], EOS, S)
                steps += 1
                assert steps < 200
            assert F == F_true
            # the end-of-audio step itself plus S - 2 further drain steps (none to flush when S <= 2)
            assert steps == max(F_true + 1, F_true + S - 1)
            D = np.array(rows, dtype=np.int64)
            for t in range(D.shape[0]):
                for i in range(S):
                    f = t - i
                    if 0 <= f < F_true:
                        assert D[t, i] == 10 * t + i
                    elif i == 0 and t == F_true:
                        assert D[t, i] == EOS            # the end-of-audio symbol itself, never part of a frame
                    else:
                        assert D[t, i] == PAD
            if S > 1 and F_true > 0:
                # S - 1 paddings on the primary stream during the drain (the EOS step aside)
                assert (D[F_true + 1:, 0] == PAD).sum() == S - 2 and D.shape[0] == F_true + S - 1
                # and the de-interleaved matrix is complete: no PAD, no EOS inside the F frames
                dl = np.full((1, F_true + S - 1, S), PAD, dtype=np.int32)
                dl[0, :D.shape[0]] = D
                grid = oracle.deinterleave(dl)[0]
                assert grid.shape == (F_true, S) and (grid != PAD).all() and (grid != EOS).all()


def test_state_machine_ignores_eos_without_an_eos_id_and_after_the_frame_count_is_set():
    assert oracle.advance_state(3, oracle.F_UNSET, 5, -1, 4) == (4, oracle.F_UNSET, False)
    assert oracle.advance_state(6, 2, 5, 5, 4) == (7, 2, True)         # F stays 2 although stream 0 shows the id again
    assert oracle.advance_state(0, oracle.F_UNSET, 5, 5, 4) == (1, 0, False)   # end of audio before any frame
