"""Pins for the oracle's arithmetic stages O1, O3, O4 (oracle/cfgms_oracle.c).

Each check ties the oracle to something other than itself: a library routine (torch bf16
casts, torch fp64 matmul), a closed form, or an identity the paper's equations fix
(PAPER.md:54 head projection, Eq. 1).
"""
import numpy as np
import pytest
import torch

import oracle
import workloads


def _bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def test_bf16_decode_all_patterns_vs_torch():
    bits = np.arange(65536, dtype=np.uint16)
    ref = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).to(torch.float64).numpy()
    got = oracle.bf16_to_f64(bits)
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan], ref[~nan])


def test_f32_to_bf16_rne_vs_torch():
    g = torch.Generator().manual_seed(1)
    x = torch.randn(200000, generator=g) * torch.exp(4 * torch.randn(200000, generator=g))
    # exact ties (lower half == 0x8000) on both parities, and the carry into the exponent
    ties = torch.from_numpy(np.array([0x3F808000, 0x3F818000, 0x3FFF8000, 0x7F7F7FFF, 0x00008000,
                                      0x80018000], dtype=np.uint32).view(np.float32))
    special = torch.tensor([0.0, -0.0, float("inf"), -float("inf"), 1e-45, 3.4e38])
    x = torch.cat([x, ties, special])
    ref = _bits(x.to(torch.bfloat16))
    got = oracle.f32_to_bf16(x.numpy())
    assert np.array_equal(got, ref)


def _small(S=3, V=20, d=48, R=6, seed=0):
    g = torch.Generator().manual_seed(seed)
    heads = (torch.randn(S, V, d, generator=g) / d ** 0.5).to(torch.bfloat16)
    embeds = (torch.randn(S, d, generator=g) * 0.14).to(torch.bfloat16)
    hidden = torch.randn(R, d, generator=g).to(torch.bfloat16)
    return heads, embeds, hidden


def test_logits_vs_torch_fp64_matmul():
    heads, embeds, hidden = _small()
    S, V, d = heads.shape
    W = heads.to(torch.float64)
    for i in range(S):
        x = hidden.to(torch.float64) + embeds[i].to(torch.float64)        # P:54  h_t + e_i
        ref = (x @ W[i].T).numpy()                                         # W_H (h_t + e_i)
        for r in range(hidden.shape[0]):
            got = oracle.logits_row(heads, embeds, hidden, r, i)
            assert np.max(np.abs(got - ref[r])) <= 1e-12 * max(1.0, np.max(np.abs(ref[r])))


def test_logits_transposed_operand_would_fail():
    # W_i is [V][d] with k contiguous: a square head whose transpose differs must not match W^T.
    g = torch.Generator().manual_seed(3)
    heads = torch.randn(1, 16, 16, generator=g).to(torch.bfloat16)
    embeds = torch.zeros(1, 16, dtype=torch.bfloat16)
    hidden = torch.randn(2, 16, generator=g).to(torch.bfloat16)
    got = oracle.logits_row(heads, embeds, hidden, 1, 0)
    ref = (hidden[1].double() @ heads[0].double().T).numpy()
    wrong = (hidden[1].double() @ heads[0].double()).numpy()
    assert np.allclose(got, ref, atol=1e-12)
    assert not np.allclose(got, wrong, atol=1e-3)


def test_logits_zero_embedding_is_plain_gemm_and_linear():
    heads, embeds, hidden = _small()
    zero = torch.zeros_like(embeds)
    for i in range(heads.shape[0]):
        lh = oracle.logits_row(heads, zero, hidden, 2, i)                 # W h
        ref = (hidden[2].double() @ heads[i].double().T).numpy()
        assert np.max(np.abs(lh - ref)) <= 1e-12
        # linearity: W(h + e) = W h + W e ; W e via a batch whose hidden row is e_i and e = 0
        le = oracle.logits_row(heads, zero, embeds, i, i)
        lhe = oracle.logits_row(heads, embeds, hidden, 2, i)
        assert np.max(np.abs(lhe - (lh + le))) <= 1e-9


def test_logits_hand_case_d1_v1():
    # d = 1, V = 1: logit = W * (h + e); bf16-exact values 1.5 * (2.0 + 0.25) = 3.375
    heads = torch.tensor([[[1.5]]], dtype=torch.bfloat16)
    embeds = torch.tensor([[0.25]], dtype=torch.bfloat16)
    hidden = torch.tensor([[2.0]], dtype=torch.bfloat16)
    assert oracle.logits_row(heads, embeds, hidden, 0, 0)[0] == 3.375


def test_logits_uses_own_stream_embedding_and_head():
    heads, embeds, hidden = _small()
    a = oracle.logits_row(heads, embeds, hidden, 0, 0)
    b = oracle.logits_row(heads, embeds, hidden, 0, 1)
    ref_b = ((hidden[0].double() + embeds[1].double()) @ heads[1].double().T).numpy()
    assert np.allclose(b, ref_b, atol=1e-12) and not np.allclose(a, b, atol=1e-3)


def test_merge_identities_eq1():
    g = np.random.default_rng(0)
    lc, lu = g.normal(size=257), g.normal(size=257)
    # north_star: w=1 reproduces the conditional logits, w=0 the unconditional ones (bit exact)
    assert np.array_equal(oracle.cfg_merge(lc, lu, 1.0), lc)
    assert np.array_equal(oracle.cfg_merge(lc, lu, 0.0), lu)
    # affine in w: M(2) = 2 M(1) - M(0);  M(w) = l_u + w (l_c - l_u) (north_star's form)
    assert np.allclose(oracle.cfg_merge(lc, lu, 2.0), 2 * lc - lu, atol=1e-13)
    assert np.allclose(oracle.cfg_merge(lc, lu, 3.5), lu + 3.5 * (lc - lu), atol=1e-12)
    # equal branches: merge is the identity for every w
    assert np.allclose(oracle.cfg_merge(lc, lc, 4.2), lc, atol=1e-13)
    # sign / swapped-operand guard at w = 3: 3 l_c - 2 l_u, not 3 l_u - 2 l_c
    assert np.allclose(oracle.cfg_merge(lc, lu, 3.0), 3 * lc - 2 * lu, atol=1e-12)


def _run(wl, t, **kw):
    return oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k,
                       wl.seed, wl.step(t), wl.req_id, wl.n_frames, wl.pad_token,
                       hidden_is_f32=wl.hidden_f32, **kw)


def test_step_merged_logits_match_torch_reference():
    wl = workloads.make_config(1)
    t = 5
    res = _run(wl, t, want_merged=True)
    hb = torch.from_numpy(oracle.f32_to_bf16(wl.hidden(t).numpy()).view(np.int16)).view(torch.bfloat16)
    H = hb.double()
    W = wl.heads.double()
    E = wl.embeds.double()
    for j, (c, i) in enumerate(res.cells):
        Lc = (H[c] + E[i]) @ W[i].T
        Lu = (H[c + 1] + E[i]) @ W[i].T
        ref = 3.0 * Lc + (1 - 3.0) * Lu
        assert np.max(np.abs(res.merged[j] - ref.numpy())) < 1e-10


def test_w1_cfg_equals_noncfg_on_cond_rows():
    # Eq. 1 at w = 1 is the conditional branch alone -> same tokens as an unpaired run of the
    # cond rows with the same req_id (invariant from PAPER.md:82 + counter-based noise)
    wl = workloads.make_config(1)
    wl.w[:] = 1.0
    off = workloads.cfg_off_twin(wl)
    for t in (3, 10):
        a = _run(wl, t)
        b = _run(off, t)
        assert np.array_equal(a.tok, b.tok)


def test_w0_cfg_equals_noncfg_on_uncond_rows():
    wl = workloads.make_config(1)
    wl.w[:] = 0.0
    a = _run(wl, 7)
    # unpaired batch made of the UNCOND rows, carrying the cond rows' parameters
    rows = torch.tensor([1, 3])
    b = oracle.step(wl.heads, wl.embeds, wl.hidden(7)[rows], torch.full((2,), -1, dtype=torch.int32),
                    wl.w[rows], wl.temp[rows], wl.top_k[rows], wl.seed, wl.step(7)[rows],
                    wl.req_id[rows], wl.n_frames[rows], wl.pad_token, hidden_is_f32=True)
    assert np.array_equal(a.tok, b.tok)


def test_companion_receives_same_token():
    wl = workloads.make_config(1)
    tokens = np.full((wl.R, wl.S), -7, dtype=np.int32)
    _run(wl, 9, tokens_out=tokens)
    assert np.array_equal(tokens[0], tokens[1]) and np.array_equal(tokens[2], tokens[3])
    assert (tokens >= 0).all() and (tokens < wl.V).all()


def test_pair_map_contract():
    assert oracle.check_pair_map(np.array([1, 0, -1, -1], dtype=np.int32)) == 0
    assert oracle.check_pair_map(np.array([-1, 2, 1, -1], dtype=np.int32)) != 0   # cond on an odd row
    assert oracle.check_pair_map(np.array([1, -1], dtype=np.int32)) != 0          # not an involution
    assert oracle.check_pair_map(np.array([3, -1, -1, 0], dtype=np.int32)) != 0   # not adjacent
    with pytest.raises(ValueError):
        wl = workloads.make_config(1)
        wl.pair_map[0] = 3
        _run(wl, 0)


def test_workload_shapes_and_layout():
    for cfg, (R, n_req) in {1: (4, 2), 2: (128, 64), 4: (384, 256)}.items():
        ov = {"d": 64, "V": 64} if cfg != 1 else None
        wl = workloads.make_config(cfg, overrides=ov)
        assert wl.R == R and wl.n_req == n_req and len(wl.head_rows()) == n_req
        assert oracle.check_pair_map(wl.pair_map) == 0
        assert wl.heads.dtype == torch.bfloat16 and wl.heads.shape == (wl.S, wl.V, wl.d)
    wl4 = workloads.make_config(4, overrides={"d": 64, "V": 64})
    assert int((wl4.pair_map >= 0).sum()) == 256 and set(wl4.top_k[wl4.head_rows()].tolist()) <= {1, 20, 50}
    assert 0 <= int(wl4.offset.min()) and int(wl4.offset.max()) < wl4.S
    w = wl4.w[wl4.head_rows()][wl4.pair_map[wl4.head_rows()] >= 0]
    assert float(w.min()) >= 1.0 and float(w.max()) <= 5.0
    # same seed -> same bits
    again = workloads.make_config(4, overrides={"d": 64, "V": 64})
    assert torch.equal(again.heads.view(torch.int16), wl4.heads.view(torch.int16))
    assert torch.equal(again.pair_map, wl4.pair_map)
