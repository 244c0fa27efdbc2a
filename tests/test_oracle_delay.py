"""Pins for the delay pattern: interleave/de-interleave identities,
PAD placement, and the step-driven delayed buffer of O5/O9."""
import numpy as np
import pytest

import oracle
import workloads


@pytest.mark.parametrize("S", [1, 2, 3, 8, 16])
@pytest.mark.parametrize("F", [1, 2, 17, 40])
def test_interleave_then_deinterleave_is_identity(S, F):
    rng = np.random.default_rng(S * 100 + F)
    grid = rng.integers(0, 1000, size=(3, F, S), dtype=np.int32)
    PAD = -5
    delayed = oracle.interleave(grid, PAD)
    assert delayed.shape == (3, F + S - 1, S)
    assert np.array_equal(oracle.deinterleave(delayed), grid)
    # delay padding: exactly S(S-1)/2 PAD cells in the first S-1 steps and again in the last S-1
    npad = S * (S - 1) // 2
    assert int((delayed == PAD).sum()) == 3 * 2 * npad
    if S > 1:
        assert int((delayed[:, : S - 1] == PAD).sum()) == 3 * npad or F < S - 1
        assert int((delayed[:, F:] == PAD).sum()) == 3 * npad or F < S - 1
    # stream i lags i steps: delayed[t][i] = grid[t - i][i]
    for i in range(S):
        assert np.array_equal(delayed[:, i:i + F, i], grid[:, :, i])


def test_deinterleave_definition_by_loops():
    rng = np.random.default_rng(9)
    T, S = 13, 4
    D = rng.integers(0, 99, size=(2, T, S), dtype=np.int32)
    G = oracle.deinterleave(D)
    assert G.shape == (2, T - S + 1, S)
    for q in range(2):
        for f in range(T - S + 1):
            for i in range(S):
                assert G[q, f, i] == D[q, f + i, i]


def test_single_stream_is_identity_copy():
    D = np.arange(2 * 7, dtype=np.int32).reshape(2, 7, 1)
    assert np.array_equal(oracle.deinterleave(D), D)


def _run_all_steps(wl, tokens_seq=None):
    delayed = np.full((wl.R, wl.T, wl.S), -1, dtype=np.int32)
    toks = []
    for t in range(wl.T):
        tokens = np.full((wl.R, wl.S), -1, dtype=np.int32)
        res = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k,
                          wl.seed, wl.step(t), wl.req_id, wl.n_frames, wl.pad_token,
                          tokens_out=tokens, delayed=delayed, hidden_is_f32=wl.hidden_f32)
        toks.append((res, tokens))
    return delayed, toks


def test_step_driven_delayed_buffer_config1():
    """BASELINE config 1 (tiny): T = 24 steps, S = 4 -> F = 21 frames."""
    wl = workloads.make_config(1)
    S, T, F, PAD = wl.S, wl.T, wl.T - wl.S + 1, wl.pad_token
    delayed, toks = _run_all_steps(wl)
    heads = wl.head_rows()
    for c in heads:
        D = delayed[c]
        for t in range(T):
            for i in range(S):
                active = i <= t < F + i
                assert (D[t, i] == PAD) == (not active)           # PAD never collides: PAD = V
                if active:
                    assert 0 <= D[t, i] < wl.V
        # PAD cells: S(S-1)/2 at the head and at the tail
        assert int((D[: S - 1] == PAD).sum()) == S * (S - 1) // 2
        assert int((D[F:] == PAD).sum()) == S * (S - 1) // 2
    # de-interleaved grid = each stream's sampled sequence re-aligned; no PAD reaches the grid
    grid = oracle.deinterleave(delayed[heads])
    assert grid.shape == (2, F, S) and (grid != PAD).all()
    for qi, c in enumerate(heads):
        for i in range(S):
            seq = [int(toks[t][1][c, i]) for t in range(i, F + i)]
            assert grid[qi, :, i].tolist() == seq
    # interleave(grid) reproduces the delayed buffer, PAD included
    assert np.array_equal(oracle.interleave(grid, PAD), delayed[heads])
    # companion rows got the same tokens every step
    for _, tokens in toks:
        assert np.array_equal(tokens[0], tokens[1]) and np.array_equal(tokens[2], tokens[3])


def test_ring_buffer_wraps_modulo_T_cap():
    wl = workloads.make_config(1)
    ring = np.full((wl.R, wl.S, wl.S), -1, dtype=np.int32)      # depth S ring
    full = np.full((wl.R, wl.T, wl.S), -1, dtype=np.int32)
    for t in range(10):
        for buf in (ring, full):
            oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k,
                        wl.seed, wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, delayed=buf,
                        hidden_is_f32=True)
    for t in range(6, 10):
        assert np.array_equal(ring[:, t % wl.S], full[:, t])


def test_determinism_under_batch_placement():
    """Counter-based noise: a request's tokens do not depend on the rows around it."""
    wl = workloads.make_config(1)
    t = 6
    a = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                    wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, hidden_is_f32=True)
    # swap the two pair slots
    perm = np.array([2, 3, 0, 1])
    sw = lambda x: x[perm]
    b = oracle.step(wl.heads, wl.embeds, wl.hidden(t)[perm], wl.pair_map, sw(wl.w), sw(wl.temp),
                    sw(wl.top_k), wl.seed, sw(wl.step(t)), sw(wl.req_id), sw(wl.n_frames), wl.pad_token,
                    hidden_is_f32=True)
    S = wl.S
    assert np.array_equal(a.tok[:S], b.tok[S:]) and np.array_equal(a.tok[S:], b.tok[:S])
    # the second request alone (R = 2)
    rows = np.array([2, 3])
    c = oracle.step(wl.heads, wl.embeds, wl.hidden(t)[rows], np.array([1, 0], dtype=np.int32),
                    wl.w[rows], wl.temp[rows], wl.top_k[rows], wl.seed, wl.step(t)[rows],
                    wl.req_id[rows], wl.n_frames[rows], wl.pad_token, hidden_is_f32=True)
    assert np.array_equal(c.tok, a.tok[S:])


def test_cell_subset_equals_full_run():
    wl = workloads.make_config(1)
    t = 4
    full = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                       wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, hidden_is_f32=True, want_merged=True)
    cells = np.array([[2, 3], [0, 1]], dtype=np.int32)
    sub = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                      wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, hidden_is_f32=True, cells=cells,
                      want_merged=True)
    assert sub.tok[0] == full.tok[wl.S + 3] and sub.tok[1] == full.tok[1]
    assert np.array_equal(sub.merged[0], full.merged[wl.S + 3])
    with pytest.raises(ValueError):   # an uncond row does not own a request
        oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                    wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, hidden_is_f32=True,
                    cells=np.array([[1, 0]], dtype=np.int32))


def test_staggered_offsets_config4_shape():
    """Reading C17: request q is at local step tau = t + o_q; at t = 0 rows with offset o have
    streams i <= o active and the rest PAD."""
    wl = workloads.make_config(4, overrides={"d": 64, "V": 64})
    res = oracle.step(wl.heads, wl.embeds, wl.hidden(0), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                      wl.step(0), wl.req_id, wl.n_frames, wl.pad_token)
    off = wl.offset.numpy()
    for (c, i), tok, fl in zip(res.cells, res.tok, res.flags):
        if i <= off[c]:
            assert 0 <= tok < wl.V and not fl & oracle.FLAG_INACTIVE
        else:
            assert tok == wl.pad_token and fl & oracle.FLAG_INACTIVE
