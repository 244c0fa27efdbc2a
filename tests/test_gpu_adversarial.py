"""Deterministic adversarial rows for the candidate sampler (K1's per-chunk top-4 pass + K2's
threshold / overflow logic), against the oracle through the C ABI.

Random Gaussian logits almost never build the situations in which the candidate path has to work
hard: a 32-token chunk holding five or more members of the top-k, a chunk whose 4th emitted value
shares the threshold's 27-bit key bucket but lies just below it, long runs of exactly equal values.
Here the temperature-scaled logits z are INSTALLED exactly: hidden states and stream embeddings are
zero (every projection is exactly 0), temperature is 1, and the crafted values enter through the
additive logit bias (cfgms_set_logit_bias), so z == bias bit for bit on both sides.  Nothing is
excused as a close tie: with z exact on both sides the 2e-2 logit tolerance does not apply, and a
token may differ from the oracle's only when the two best perturbed scores are within 1e-4 (the fp32
noise evaluation), and then only by a token that could have won (parity_util.valid_alternative)."""
import numpy as np
import pytest
import torch

import oracle
import workloads
from parity_util import DeviceWorkload, valid_alternative

pytestmark = pytest.mark.gpu

V = 2048
NOISE_TOL = 1e-4     # fp32 vs fp64 evaluation of z + g (see the comparison loop)


def _lows(rng):
    """Distinct, clearly losing values for the rest of the vocabulary."""
    return (-30.0 - 1e-3 * rng.permutation(V)).astype(np.float32)


def _row_straddle(rng):
    """The advisor's row: chunk A = {13.0, 12.95, 12.9, t - 1ulp}, chunk B = five top values, chunk C = {t}.
    With k = 8 the 8th largest EMITTED value is t, but the true threshold is 12.9: chunk B hides its fifth
    value, and chunk A's 4th emitted value sits in t's key bucket, just below t."""
    z = _lows(rng)
    t = np.float32(12.8)
    assert (t.view(np.uint32) & 31) != 0            # t - 1ulp shares t's 27-bit key bucket
    z[3 * 32 + np.array([1, 9, 17, 30])] = [13.0, 12.95, 12.9, np.nextafter(t, np.float32(-np.inf))]
    z[10 * 32 + np.array([0, 3, 11, 20, 31])] = [13.4, 13.3, 13.2, 13.1, 13.05]
    z[20 * 32 + 7] = t
    return z


def _row_many_ties(rng):
    """300 exactly equal maxima (more than the sampler's candidate list holds): threshold semantics keeps
    them all, the candidate path must fall back to the full-row scan."""
    z = _lows(rng)
    z[np.arange(300) * 6 + 2] = 5.0
    return z


def _row_one_hot_chunk(rng):
    """Twelve of the top values inside ONE chunk: only four are emitted, the 8th largest emitted value is a
    'low' one, and the exact threshold has to come from the re-read chunk."""
    z = _lows(rng)
    z[5 * 32 + np.arange(4, 28, 2)] = np.linspace(10.0, 11.0, 12, dtype=np.float32)
    return z


def _row_ties_at_the_edge(rng):
    """Twenty equal values at the top with k = 8: all twenty tie at the k-th place and stay."""
    z = _lows(rng)
    z[rng.choice(V, size=20, replace=False)] = 7.25
    return z


def _row_bucket_neighbours(rng):
    """Values that differ by single ulps around the k-th place, spread over chunks: the 27-bit bucket
    bound must never drop or admit one of them wrongly."""
    z = _lows(rng)
    base = np.float32(9.0)
    vals = [base]
    for _ in range(11):
        vals.append(np.nextafter(vals[-1], np.float32(-np.inf)))
    pos = rng.choice(V, size=12, replace=False)
    z[pos] = np.asarray(vals, dtype=np.float32)
    z[rng.choice(np.setdiff1d(np.arange(V), pos), size=3, replace=False)] = [9.5, 9.4, 9.3]
    return z


ROWS = [_row_straddle, _row_many_ties, _row_one_hot_chunk, _row_ties_at_the_edge, _row_bucket_neighbours]


@pytest.mark.parametrize("top_k", [8, 1, 12])
def test_crafted_rows_candidate_sampler_is_exact(top_k):
    dev = torch.device("cuda:0")
    S = len(ROWS)
    wl = workloads.make_config(2, overrides=dict(pairs=24, singles=16, d=64, S=S, V=V, T=S + 20, top_k=top_k, temp=1.0,
                                                 hidden_f32=False, heavy_tail=False))
    wl.hidden_pool.zero_()
    wl.embeds.zero_()
    rng = np.random.default_rng(77)
    bias = np.stack([f(rng) for f in ROWS]).astype(np.float32)
    dw = DeviceWorkload(wl, dev)
    assert dw.ctx.info()["V"] == V
    dw.ctx.set_logit_bias(torch.from_numpy(bias).to(dev))
    pm = wl.pair_map.numpy()
    n_sampled = n_close = n_diff = 0
    for t in (S, S + 1, S + 2):
        logits = torch.full((wl.R, S, V), 1.0, dtype=torch.float32, device=dev)
        dw.tokens.fill_(-1)
        dw.step(t, logits_out=logits)
        dw.check_no_device_error()
        ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                          wl.req_id, wl.n_frames, wl.pad_token, want_merged=True, logit_bias=bias.astype(np.float64))
        got, gl = dw.tokens.cpu().numpy(), logits.cpu().numpy()
        for j, (c, i) in enumerate(ref.cells):
            assert not (ref.flags[j] & oracle.FLAG_INACTIVE)
            assert np.array_equal(gl[c, i], bias[i]) and np.array_equal(ref.merged[j], bias[i].astype(np.float64))   # z installed exactly
            if pm[c] >= 0:
                assert got[pm[c], i] == got[c, i]
            n_sampled += 1
            # z carries NO error here, so the oracle's close / boundary flags (which allow for 2e-2 of logit
            # error) excuse nothing: the only difference left between the two sides is the fp32 evaluation of
            # the Gumbel noise (abs. error < 1e-5), so tokens must agree unless the
            # oracle's best-minus-second perturbed score is below 1e-4 — and then the token must still be one
            # that could have won.
            if ref.margin[j] <= NOISE_TOL and not (ref.flags[j] & oracle.FLAG_GREEDY):   # greedy: no noise, lowest index among equals
                n_close += 1
                if got[c, i] != ref.tok[j]:
                    n_diff += 1
                    assert valid_alternative(wl, t, c, i, int(got[c, i]), logit_bias=bias, tol=NOISE_TOL), (t, c, i)
            else:
                assert got[c, i] == ref.tok[j], (top_k, t, c, i, ROWS[i].__name__, got[c, i], ref.tok[j], ref.margin[j])
    print(f"adversarial rows, top_k={top_k}: {n_sampled} cells, {n_close} with margin <= {NOISE_TOL}, {n_diff} of them differ")
    assert n_diff <= n_close <= 0.01 * n_sampled + 1
    # the full-scan sampler (no candidate pass) gives the same tokens
    full = DeviceWorkload(wl, dev, no_candidates=True)
    full.ctx.set_logit_bias(torch.from_numpy(bias).to(dev))
    for t in (S, S + 2):
        dw.step(t)
        full.step(t)
        torch.cuda.synchronize()
        assert torch.equal(dw.tokens, full.tokens)
