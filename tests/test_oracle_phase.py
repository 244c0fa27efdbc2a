"""Pins of the oracle's phase state machine (widening W6; readings C28-C32):
hand-written traces of the transition function, and the phase-aware step against special cases that
reduce to the already pinned oracle.step (all-audio batch; merge bypass == a non-CFG run; a vocabulary
region == -inf masking of its complement; modality == numpy argmax)."""
import numpy as np
import pytest

import oracle
import workloads
from oracle import F_UNSET, PHASE_AUDIO as A, PHASE_DONE as D, PHASE_TEXT as T, PHASE_TRANSITION as X


def test_transition_function_hand_traces():
    S, eos, nb = 4, 99, 3
    adv = lambda ph, pos, F, tok0=5, mod=False: oracle.phase_advance(ph, pos, F, tok0, mod, nb, eos, S)
    # text phase: stays while the model asks for text, whatever token it emitted (even the audio-side eos id)
    assert adv(T, 0, F_UNSET) == (T, 0, F_UNSET, False)
    assert adv(T, 7, F_UNSET, tok0=eos) == (T, 0, F_UNSET, False)
    # the step on which the unmasked argmax falls into the audio region ends the text phase (C29)
    assert adv(T, 0, F_UNSET, mod=True) == (X, 0, F_UNSET, False)
    # three bridging tokens, then audio-local step 0 (C30)
    assert adv(X, 0, F_UNSET) == (X, 1, F_UNSET, False)
    assert adv(X, 1, F_UNSET) == (X, 2, F_UNSET, False)
    assert adv(X, 2, F_UNSET, mod=True) == (A, 0, F_UNSET, False)
    # audio: tau_a counts up; the end-of-audio token at tau_a = 6 fixes F = 6 (C27/C31)
    assert adv(A, 0, F_UNSET) == (A, 1, F_UNSET, False)
    assert adv(A, 6, F_UNSET, tok0=eos) == (A, 7, 6, False)
    # drain: S - 1 = 3 more steps (tau_a = 7, 8 end at 9 >= 6 + 3)
    assert adv(A, 7, 6) == (A, 8, 6, False)
    assert adv(A, 8, 6, tok0=eos) == (D, 9, 6, True)        # a second eos changes nothing
    assert adv(D, 9, 6) == (D, 9, 6, True)                  # frozen
    # a frame count given from outside drains the same way
    assert adv(A, 4, 3) == (A, 5, 3, False) and adv(A, 5, 3) == (D, 6, 3, True)      # 6 >= F + S - 1
    # no bridging tokens configured: text -> audio directly
    assert oracle.phase_advance(T, 0, F_UNSET, 5, True, 0, eos, S) == (A, 0, F_UNSET, False)
    # no end-of-audio id: the frame count never sets itself
    assert oracle.phase_advance(A, 3, F_UNSET, 99, False, nb, -1, S) == (A, 4, F_UNSET, False)


def test_a_request_driven_through_all_phases_counts_its_steps():
    """text steps + n_bridge + (F + S - 1) audio steps; stream 0 pads S - 1 times in the drain."""
    S, eos, nb = 5, 7, 2
    for t_switch, t_eos in ((0, 0), (3, 4), (1, 11)):
        ph, pos, F, steps, trace = T, 0, F_UNSET, 0, []
        while ph != D and steps < 100:
            tok0 = eos if (ph == A and pos == t_eos) else 1
            mod = ph == T and steps == t_switch
            trace.append(ph)
            ph, pos, F, done = oracle.phase_advance(ph, pos, F, tok0, mod, nb, eos, S)
            steps += 1
        assert trace.count(T) == t_switch + 1 and trace.count(X) == nb
        assert F == t_eos and trace.count(A) == max(t_eos + S - 1, 1) and done


def _wl(**kw):
    ov = dict(pairs=3, singles=2, d=128, S=4, V=256, T=24, mixed=True, hidden_f32=False, heavy_tail=False)
    ov.update(kw)
    return workloads.make_config(4, overrides=ov)


def _step_phase(wl, t, phase, pos, V_text, bridge, gstep=None, **kw):
    gs = wl.step(t) if gstep is None else gstep
    return oracle.step_phase(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, gs,
                             phase, pos, V_text, bridge, req_id=wl.req_id, n_frames=wl.n_frames, pad_token=wl.pad_token,
                             want_merged=True, **kw)


def test_all_audio_batch_equals_the_plain_step_bit_for_bit():
    wl = _wl()
    for t in (0, 2, 9):
        tau = wl.step(t)
        ph = np.full(wl.R, A, dtype=np.int32)
        a = _step_phase(wl, t, ph, tau.numpy(), 0, [])
        b = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, tau, wl.req_id,
                        wl.n_frames, wl.pad_token, want_merged=True)
        assert np.array_equal(a.tok, b.tok) and np.array_equal(a.flags, b.flags)
        assert np.array_equal(a.margin, b.margin) and np.array_equal(a.merged, b.merged)
        assert not a.modality.any()


def test_text_phase_bypasses_the_merge_and_restricts_stream0_to_the_text_region():
    wl = _wl(pairs=5, singles=2)
    V_text = 96
    t = 6
    ph = np.full(wl.R, T, dtype=np.int32)
    got = _step_phase(wl, t, ph, np.zeros(wl.R, dtype=np.int32), V_text, [1, 2])
    # reference: the CFG-off twin (cond rows only, every row its own request: NO merge) with the audio region of
    # stream 0 masked by -inf through the already pinned W2 bias
    off = workloads.cfg_off_twin(wl)
    bias = np.zeros((wl.S, wl.V))
    bias[0, V_text:] = -np.inf
    ref = oracle.step(off.heads, off.embeds, off.hidden(t), off.pair_map, off.w, off.temp, off.top_k, off.seed, off.step(t),
                      off.req_id, None, off.pad_token, want_merged=True, logit_bias=bias)
    heads = wl.head_rows()
    row_of = {int(c): q for q, c in enumerate(heads)}
    for j, (c, i) in enumerate(got.cells):
        k = row_of[int(c)] * wl.S + int(i)
        assert tuple(ref.cells[k]) == (row_of[int(c)], i)
        if i == 0:
            assert got.tok[j] == ref.tok[k] and 0 <= got.tok[j] < V_text
            # cond-only logits, unmasked: the twin's merged row before the mask
            unmasked = ref.merged[k].copy()
            unmasked[V_text:] = oracle.logits_row(wl.heads, wl.embeds, wl.hidden(t), int(c), 0)[V_text:]
            assert np.array_equal(got.merged[j], unmasked)
            assert got.modality[j] == int(np.argmax(got.merged[j]) >= V_text)       # C29 vs numpy
        else:
            assert got.tok[j] == wl.pad_token and got.flags[j] & oracle.FLAG_INACTIVE and got.modality[j] == 0
    assert 0 < got.modality[got.cells[:, 1] == 0].sum() < len(heads)      # both modalities occur in this batch


def test_audio_phase_region_equals_masking_the_text_region():
    wl = _wl()
    V_text = 64
    t = 9
    tau = wl.step(t)
    ph = np.full(wl.R, A, dtype=np.int32)
    got = _step_phase(wl, t, ph, tau.numpy(), V_text, [3])
    bias = np.zeros((wl.S, wl.V))
    bias[0, :V_text] = -np.inf
    ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, tau, wl.req_id,
                      wl.n_frames, wl.pad_token, logit_bias=bias)
    assert np.array_equal(got.tok, ref.tok)
    s0 = got.cells[:, 1] == 0
    assert (got.tok[s0 & (got.flags & oracle.FLAG_INACTIVE == 0)] >= V_text).all()


def test_transition_and_done_phases_sample_nothing():
    wl = _wl()
    bridge = [250, 3, 77]
    ph = np.asarray([X, X, A, A, D, D, T, T, X, X][:wl.R], dtype=np.int32)
    pos = np.asarray([0, 0, 2, 2, 5, 5, 0, 0, 2, 2][:wl.R], dtype=np.int32)
    got = _step_phase(wl, 4, ph, pos, 128, bridge, gstep=np.full(wl.R, 40, dtype=np.int32))
    for j, (c, i) in enumerate(got.cells):
        if ph[c] == X:
            assert got.tok[j] == (bridge[pos[c]] if i == 0 else wl.pad_token)
            assert got.flags[j] == (oracle.FLAG_FORCED if i == 0 else oracle.FLAG_INACTIVE)
        if ph[c] == D:
            assert got.tok[j] == wl.pad_token and got.flags[j] == oracle.FLAG_INACTIVE
        if ph[c] == A:       # audio-local step 2: streams 0..2 active, stream 3 not yet
            assert (got.flags[j] & oracle.FLAG_INACTIVE != 0) == (i > 2)


def test_noise_is_keyed_by_the_global_step_not_the_phase_position():
    """C32: the same audio-local position reached at different global steps draws different noise; and the
    phase-aware step with gstep == pos reproduces the plain step (covered above)."""
    wl = _wl(pairs=4, singles=0)
    ph = np.full(wl.R, A, dtype=np.int32)
    pos = np.full(wl.R, 7, dtype=np.int32)
    a = _step_phase(wl, 7, ph, pos, 0, [], gstep=np.full(wl.R, 7, dtype=np.int32))
    b = _step_phase(wl, 7, ph, pos, 0, [], gstep=np.full(wl.R, 19, dtype=np.int32))
    assert np.array_equal(a.merged, b.merged) and not np.array_equal(a.tok, b.tok)
    plain = oracle.step(wl.heads, wl.embeds, wl.hidden(7), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, pos, wl.req_id,
                        wl.n_frames, wl.pad_token)
    assert np.array_equal(a.tok, plain.tok)
