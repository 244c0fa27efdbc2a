"""Host logic of the GPU parity harness (no GPU needed): the valid-alternative rule applied to
close ties, and the bound on how many cells may be close."""
import numpy as np
import pytest

import oracle
import workloads
from parity_util import ParityStats, sample_cells, valid_alternative


def test_valid_alternative_accepts_the_oracle_token_and_rejects_losers():
    wl = workloads.make_config(1)
    t = 7
    ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                      wl.req_id, wl.n_frames, wl.pad_token, want_merged=True, hidden_is_f32=True)
    for j, (c, i) in enumerate(ref.cells):
        assert valid_alternative(wl, t, c, i, int(ref.tok[j]))
        z = ref.merged[j] / float(wl.temp[c])
        loser = int(np.argmin(z))                        # far outside the top-16
        assert not valid_alternative(wl, t, c, i, loser)
        assert not valid_alternative(wl, t, c, i, wl.V)  # not a token at all
        # a survivor whose perturbed score trails the winner by more than 2 * tol is no alternative
        thr = np.sort(z)[::-1][int(wl.top_k[c]) - 1]
        g = np.array([oracle.gumbel(wl.seed, int(wl.req_id[c]), int(wl.step(t)[c]), int(i), v) for v in range(wl.V)])
        s = np.where(z >= thr, z + g, -np.inf)
        order = np.argsort(s)[::-1]
        assert order[0] == ref.tok[j]
        far = [int(v) for v in order[1:] if np.isfinite(s[v]) and s[order[0]] - s[v] > 0.05]
        near = [int(v) for v in order[1:] if np.isfinite(s[v]) and s[order[0]] - s[v] < 0.03]
        assert far and not valid_alternative(wl, t, c, i, far[0])
        for v in near:
            assert valid_alternative(wl, t, c, i, v)


def test_valid_alternative_greedy_and_bias():
    wl = workloads.make_config(1)
    wl.top_k[:] = 1
    t = 5
    c, i = int(wl.head_rows()[0]), 2
    ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                      wl.req_id, wl.n_frames, wl.pad_token, cells=[(c, i)], want_merged=True, hidden_is_f32=True)
    best = int(ref.tok[0])
    assert valid_alternative(wl, t, c, i, best)
    second = int(np.argsort(ref.merged[0])[::-1][1])
    assert valid_alternative(wl, t, c, i, second) == bool(ref.merged[0][best] - ref.merged[0][second] <= 0.04)
    bias = np.zeros((wl.S, wl.V))
    bias[i, second] = 100.0                              # with the bias the runner-up wins outright
    assert valid_alternative(wl, t, c, i, second, logit_bias=bias)
    assert not valid_alternative(wl, t, c, i, best, logit_bias=bias)


def test_close_fraction_bound():
    st = ParityStats()
    st.n, st.n_pad, st.n_close, st.n_close_mismatch = 1000, 100, 20, 1
    st.assert_close_fraction()                           # 20 <= 0.03 * 900 + 2
    st.n_close = 40
    with pytest.raises(AssertionError):
        st.assert_close_fraction()
    st.n_close, st.n_close_mismatch = 3, 4
    with pytest.raises(AssertionError):
        st.assert_close_fraction()


def test_sample_cells_is_seeded_and_owns_requests():
    wl = workloads.make_config(4)
    a, b = sample_cells(wl, 50, seed=3), sample_cells(wl, 50, seed=3)
    assert np.array_equal(a, b) and len(a) == 50
    heads = set(wl.head_rows().tolist())
    assert all(int(r) in heads and 0 <= int(i) < wl.S for r, i in a)
    assert len(sample_cells(wl, None, seed=0)) == wl.n_req * wl.S
