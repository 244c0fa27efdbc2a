"""GPU parity of the widenings against the oracle, through the C ABI:
W1 streaming frame emission (bit-exact), W2 static logit bias + forced tokens (same tolerance
rules as the main path), W3 feedback aggregation (correctly rounded bf16 of the exact sum),
W4 device-resident request state with automatic drain (bit-exact), W5 stream-sharded heads
(shards merged == unsharded, bit-exact)."""
import numpy as np
import pytest
import torch

import oracle
import workloads
from parity_util import LOGIT_TOL, DeviceWorkload, check_tokens_against_oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    return torch.device("cuda:0")


def _custom(pairs, singles, d, S, V, T=16, mixed=False, **kw):
    ov = dict(pairs=pairs, singles=singles, d=d, S=S, V=V, T=T, mixed=mixed, hidden_f32=False, heavy_tail=False)
    ov.update(kw)
    return workloads.make_config(2 if not mixed else 4, overrides=ov)


# ------------------------------------------------------------------ W1
@pytest.mark.parametrize("case", [
    dict(wl=("config", 1), T_cap=None, no_candidates=False),          # full delayed matrix
    dict(wl=("config", 1), T_cap=4, no_candidates=False),             # ring of depth exactly S
    dict(wl=("config", 1), T_cap=7, no_candidates=True),              # full-scan sampler kernel
    dict(wl=("custom", dict(pairs=3, singles=4, d=128, S=9, V=160, T=30)), T_cap=9, no_candidates=False),
    dict(wl=("custom", dict(pairs=1, singles=2, d=64, S=1, V=64, T=6)), T_cap=1, no_candidates=False),
])
def test_streaming_frames_equal_the_deinterleaved_grid(dev, case):
    kind, arg = case["wl"]
    wl = workloads.make_config(arg) if kind == "config" else _custom(**arg)
    dw = DeviceWorkload(wl, dev, T_cap=case["T_cap"], no_candidates=case["no_candidates"])
    full = DeviceWorkload(wl, dev)                  # keeps the whole delayed matrix for the bulk de-interleave
    R, S, pad = wl.R, wl.S, wl.pad_token
    nf = wl.n_frames.numpy() if wl.n_frames is not None else None
    heads = wl.head_rows()
    pm = wl.pair_map.numpy()
    frames = {int(c): {} for c in heads}
    for t in range(wl.T):
        frame = torch.full((R, S), -9, dtype=torch.int32, device=dev)
        fidx = torch.full((R,), -9, dtype=torch.int32, device=dev)
        st = wl.step(t).to(dev)
        dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, st, dw.tokens, req_id=dw.req_id,
                    n_frames=dw.n_frames, delayed=dw.delayed, frame_out=frame, frame_index_out=fidx)
        full.step(t)
        dw.check_no_device_error()
        fr, fi, ring = frame.cpu().numpy(), fidx.cpu().numpy(), dw.delayed.cpu().numpy()
        tau = wl.step(t).numpy()
        for c in heads:
            # the oracle's emission rule applied to the GPU's own ring (integer work: bit-exact)
            want_f, want_fr = oracle.emit_frame(ring[c], int(tau[c]), int(nf[c]) if nf is not None else -1, pad)
            assert fi[c] == want_f and np.array_equal(fr[c], want_fr), (t, c)
            if want_f >= 0:
                frames[int(c)][want_f] = fr[c].copy()
            if pm[c] >= 0:      # companion outputs stay hidden
                assert fi[pm[c]] == -1 and np.all(fr[pm[c]] == pad)
    # all frames of a request, in order, are exactly the bulk de-interleave of its delayed matrix
    grid = oracle.deinterleave(full.delayed.cpu().numpy()[heads])
    for q, c in enumerate(heads):
        F = grid.shape[1] if nf is None else min(int(nf[c]), grid.shape[1])
        got = frames[int(c)]
        tau0 = int(wl.step(0).numpy()[c])
        want_ids = [f for f in range(F) if tau0 <= f + S - 1 < tau0 + wl.T]      # frames completing inside the window
        assert sorted(got) == want_ids
        if tau0 == 0:
            for f in want_ids:
                assert np.array_equal(got[f], grid[q, f]), (c, f)


def test_frame_emission_needs_a_ring_of_depth_S(dev):
    import paper_2607_02119_b200 as pkg
    wl = workloads.make_config(1)
    dw = DeviceWorkload(wl, dev, T_cap=2)
    frame = torch.zeros((wl.R, wl.S), dtype=torch.int32, device=dev)
    with pytest.raises(pkg.CfgmsError) as e:
        dw.ctx.step(dw.hidden(0), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, wl.step(0).to(dev), dw.tokens,
                    delayed=dw.delayed, frame_out=frame)
    assert e.value.status == 1      # CFGMS_ERR_ARG


# ------------------------------------------------------------------ W2
def _compare_ext(dw, t, logit_bias=None, force_token=None):
    """One GPU step with the widening inputs against oracle.step(...) with the same inputs."""
    wl, dev = dw.wl, dw.dev
    logits = torch.zeros((wl.R, wl.S, wl.V), dtype=torch.float32, device=dev)
    dw.tokens.fill_(-1)
    ft_dev = None if force_token is None else torch.from_numpy(force_token).to(dev)
    dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, wl.step(t).to(dev), dw.tokens,
                req_id=dw.req_id, n_frames=dw.n_frames, delayed=dw.delayed, logits_out=logits, force_token=ft_dev)
    dw.check_no_device_error()
    ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                      wl.req_id, wl.n_frames, wl.pad_token, want_merged=True, hidden_is_f32=wl.hidden_f32,
                      logit_bias=logit_bias, force_token=force_token)
    got, gl = dw.tokens.cpu().numpy(), logits.cpu().numpy().astype(np.float64)
    pm = wl.pair_map.numpy()
    n_close = n_forced = 0
    for j, (c, i) in enumerate(ref.cells):
        fl = int(ref.flags[j])
        if pm[c] >= 0:
            assert got[pm[c], i] == got[c, i]
        if fl & oracle.FLAG_INACTIVE:
            assert got[c, i] == wl.pad_token
        elif fl & oracle.FLAG_FORCED:
            n_forced += 1
            assert got[c, i] == force_token[c, i]
        else:
            m = ref.merged[j]
            fin = np.isfinite(m)
            assert np.array_equal(np.isneginf(gl[c, i]), np.isneginf(m))          # masked tokens are -inf on both sides
            assert np.max(np.abs(gl[c, i][fin] - m[fin])) <= LOGIT_TOL
            if fl & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
                n_close += 1
            else:
                assert got[c, i] == ref.tok[j], (t, c, i, got[c, i], ref.tok[j], ref.margin[j])
            assert np.isfinite(m[got[c, i]])                                        # never a masked token
    return n_close, n_forced


@pytest.mark.parametrize("no_candidates", [False, True])
def test_logit_bias_masks_and_forced_tokens(dev, no_candidates):
    wl = _custom(pairs=6, singles=4, d=256, S=4, V=512, T=16, mixed=True, top_k=20)
    dw = DeviceWorkload(wl, dev, no_candidates=no_candidates)
    rng = np.random.default_rng(12)
    bias = rng.normal(scale=0.5, size=(wl.S, wl.V))
    bias[0, 100:] = -np.inf                     # stream 0 may only use its first 100 tokens (< top_k survivors stay finite)
    bias[1, rng.random(wl.V) < 0.5] = -np.inf   # scattered mask
    bias[2, 7:] = -np.inf                       # 7 tokens left: fewer than top_k
    bias[3, :] = 0.0
    ft = np.full((wl.R, wl.S), -1, dtype=np.int32)
    for c in wl.head_rows()[::3]:
        ft[c, 1] = 300 + int(c)                 # bridging token on stream 1
        ft[c, 3] = wl.pad_token                 # text-phase padding on stream 3
    dw.ctx.set_logit_bias(torch.from_numpy(bias.astype(np.float32)).to(dev))
    bias32 = bias.astype(np.float32).astype(np.float64)      # the oracle sees the same fp32 values
    n_forced = 0
    for t in (0, 2, 5, 9):
        _, nf = _compare_ext(dw, t, logit_bias=bias32, force_token=ft)
        n_forced += nf
    assert n_forced > 0
    # clearing the bias restores the plain path
    dw.ctx.set_logit_bias(None)
    _compare_ext(dw, 5)


def test_logit_bias_on_config2_shape_in_the_bench_launch_configuration(dev):
    wl = workloads.make_config(2)
    dw = DeviceWorkload(wl, dev)
    rng = np.random.default_rng(3)
    bias = np.where(rng.random((wl.S, wl.V)) < 0.3, -np.inf, 0.0) + rng.normal(scale=0.2, size=(wl.S, wl.V))
    dw.ctx.set_logit_bias(torch.from_numpy(bias.astype(np.float32)).to(dev))
    n_close, _ = _compare_ext(dw, 40, logit_bias=bias.astype(np.float32).astype(np.float64))
    assert n_close < 0.08 * wl.n_req * wl.S


# ------------------------------------------------------------------ W3
def _bf16_ulp(x):
    """Spacing of bf16 (8 significand bits) at |x| (float64 array)."""
    ax = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)


@pytest.mark.parametrize("shape", [
    dict(R=7, S=3, V_e=50, d=64),            # odd row count, one 16-byte chunk per 8 columns
    dict(R=64, S=9, V_e=257, d=2048),        # OpusLM-like 9 streams
    dict(R=256, S=16, V_e=2049, d=4096),     # config-5 head shape (V + 1 rows: PAD has an embedding)
    dict(R=9, S=20, V_e=33, d=1096),         # more streams than one round of gathers holds; a ragged column count
    dict(R=1, S=64, V_e=5, d=8),             # one row, the most streams the head takes, one chunk
    dict(R=33, S=20, V_e=33, d=1096),        # odd row count, three rounds of gathers, a slot whose rows differ
    dict(R=40, S=64, V_e=9, d=512),          # the most streams the head takes, many rows
    dict(R=700, S=3, V_e=11, d=4096),        # more slots than two waves of CTAs, few streams, wide rows
])
def test_feedback_is_the_correctly_rounded_sum(dev, shape):
    R, S, V_e, d = shape["R"], shape["S"], shape["V_e"], shape["d"]
    g = torch.Generator().manual_seed(R + S)
    emb = (torch.randn(S, V_e, d, generator=g) * 0.5).to(torch.bfloat16)
    tok = torch.randint(0, V_e, (R, S), generator=g, dtype=torch.int32)
    tok[1::2] = tok[0::2][: tok[1::2].shape[0]]          # companion rows carry their cond row's tokens
    if R > 4:
        tok[4, 0] = -1                                    # ids outside [0, V_e) contribute nothing
        tok[4, S - 1] = V_e
        tok[3, 1] = (tok[3, 1] + 1) % V_e                 # a slot whose two rows differ
    heads = torch.zeros(S, 128, d, dtype=torch.bfloat16, device=dev)
    import paper_2607_02119_b200 as pkg
    ctx = pkg.Context(heads, torch.zeros(S, d, dtype=torch.bfloat16, device=dev), max_rows=8)
    x = ctx.feedback(tok.to(dev), emb.to(dev))
    torch.cuda.synchronize()
    got = x.float().cpu().numpy().astype(np.float64)
    want = oracle.feedback(tok.numpy(), emb)
    # fp32 accumulation of S bf16 terms then one RNE to bf16: within half a bf16 ulp of the exact sum,
    # plus the fp32 accumulation error (S * 2^-24 * sum of |terms| <= S * 2^-24 * S * max|term|)
    terms_max = float(emb.float().abs().max())
    tol = 0.5 * _bf16_ulp(want) * (1 + 1e-6) + S * S * 2.0 ** -24 * terms_max
    assert np.all(np.abs(got - want) <= tol), float(np.max(np.abs(got - want) / _bf16_ulp(want)))
    assert np.array_equal(got[1][: d], got[0][: d]) if R >= 2 else True
    ctx.close()


# ------------------------------------------------------------------ W4
def test_device_resident_state_drives_requests_through_drain(dev):
    """Self-driving decode loop: step / frame-count state ping-pongs between two device buffers, the
    end-of-audio token on stream 0 (injected per request at a different step through force_token) fixes
    the frame count, drain follows, done flags rise; frame emission (W1) hands out exactly F frames.
    Every step is compared with the oracle driven by oracle.advance_state on the host."""
    wl = _custom(pairs=3, singles=2, d=128, S=4, V=256, T=40, mixed=True)
    wl.temp[:] = 0.0                       # greedy: no close ties to excuse, tokens must match exactly
    dw = DeviceWorkload(wl, dev, T_cap=wl.S)
    R, S, EOS = wl.R, wl.S, wl.V - 1
    heads = [int(c) for c in wl.head_rows()]
    eos_at = {c: 3 + 4 * k for k, c in enumerate(heads)}
    eos_at[heads[-1]] = 10 ** 6            # the last request never ends inside the window
    UNSET = oracle.F_UNSET
    st = [torch.zeros(R, dtype=torch.int32, device=dev), torch.zeros(R, dtype=torch.int32, device=dev)]
    nf = [torch.full((R,), UNSET, dtype=torch.int32, device=dev), torch.full((R,), UNSET, dtype=torch.int32, device=dev)]
    done = torch.zeros(R, dtype=torch.int32, device=dev)
    frame = torch.zeros((R, S), dtype=torch.int32, device=dev)
    fidx = torch.zeros(R, dtype=torch.int32, device=dev)
    o_tau = {c: 0 for c in heads}
    o_F = {c: UNSET for c in heads}
    n_frames_emitted = {c: 0 for c in heads}
    for t in range(30):
        ft = np.full((R, S), -1, dtype=np.int32)
        for c in heads:
            if o_tau[c] == eos_at[c]:
                ft[c, 0] = EOS
        a, b = st[t & 1], st[(t + 1) & 1]
        fa, fb = nf[t & 1], nf[(t + 1) & 1]
        dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, a, dw.tokens, req_id=dw.req_id,
                    n_frames=fa, delayed=dw.delayed, force_token=torch.from_numpy(ft).to(dev), frame_out=frame,
                    frame_index_out=fidx, eos_token=EOS, step_next_out=b, n_frames_next_out=fb, done_out=done)
        dw.check_no_device_error()
        # the oracle, driven by its own state
        o_step = np.zeros(R, dtype=np.int32)
        o_nf = np.full(R, UNSET, dtype=np.int32)
        for c in heads:
            o_step[c], o_nf[c] = o_tau[c], o_F[c]
        ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, o_step,
                          wl.req_id, o_nf, wl.pad_token, force_token=ft)
        got = dw.tokens.cpu().numpy()
        tok0 = {}
        for j, (c, i) in enumerate(ref.cells):
            assert got[c, i] == ref.tok[j], (t, c, i)
            if i == 0:
                tok0[int(c)] = int(ref.tok[j])
        g_step, g_nf, g_done, g_fidx = b.cpu().numpy(), fb.cpu().numpy(), done.cpu().numpy(), fidx.cpu().numpy()
        for c in heads:
            o_tau[c], o_F[c], d = oracle.advance_state(o_tau[c], o_F[c], tok0[c], EOS, S)
            assert (g_step[c], g_nf[c], bool(g_done[c])) == (o_tau[c], o_F[c], d), (t, c)
            if g_fidx[c] >= 0:
                assert g_fidx[c] == n_frames_emitted[c]        # frames come out in order, none twice
                n_frames_emitted[c] += 1
    for c in heads[:-1]:
        assert o_F[c] == eos_at[c] and n_frames_emitted[c] == o_F[c]      # exactly F frames were handed out
    assert o_F[heads[-1]] == UNSET


# ------------------------------------------------------------------ W5: stream-sharded heads
@pytest.mark.parametrize("world", [2, 3])
def test_stream_sharded_contexts_sample_what_the_unsharded_head_samples(dev, world):
    """Each 'rank' (here: independent contexts on one GPU, launched one after the other — no kernel waits
    on another) holds the head slices of streams {g, g + G, ...} with stream_base / stream_stride;
    merged, their tokens must equal the unsharded context's bit for bit (counter-based noise keyed by
    the GLOBAL stream, delay pattern on the global stream index), PAD cells included."""
    import paper_2607_02119_b200 as pkg
    from paper_2607_02119_b200 import dist_utils
    wl = _custom(pairs=5, singles=2, d=256, S=9, V=256, T=24, mixed=True)       # OpusLM-like 9 streams
    full = DeviceWorkload(wl, dev)
    R, S = wl.R, wl.S
    shards = []
    for g in range(world):
        base, stride, s_local = dist_utils.stream_shard(g, world, S)
        heads = wl.heads[base::stride].contiguous().to(dev)
        embeds = wl.embeds[base::stride].contiguous().to(dev)
        assert heads.shape[0] == s_local
        ctx = pkg.Context(heads, embeds, max_rows=R, stream_base=base, stream_stride=stride)
        shards.append((ctx, heads, embeds, torch.full((R, s_local), -1, dtype=torch.int32, device=dev)))
    for t in (0, 1, 4, 8, 9, 15, 23):
        full.step(t)
        st = wl.step(t).to(dev)
        for ctx, _, _, tok in shards:
            ctx.step(full.hidden(t), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, tok,
                     req_id=full.req_id, n_frames=full.n_frames)
        torch.cuda.synchronize()
        merged = dist_utils.merge_stream_shards([s[3] for s in shards], S)
        assert torch.equal(merged, full.tokens), t
        check_tokens_against_oracle(wl, t, merged.cpu().numpy())      # and not only equal to another CUDA context
    # a frame needs every stream: sharded contexts refuse frame emission
    fr = torch.zeros((R, shards[1][3].shape[1]), dtype=torch.int32, device=dev)
    dl = torch.zeros((R, 16, shards[1][3].shape[1]), dtype=torch.int32, device=dev)
    with pytest.raises(pkg.CfgmsError) as e:
        shards[1][0].step(full.hidden(0), full.pair_map, full.w, full.temp, full.top_k, wl.seed, wl.step(0).to(dev),
                          shards[1][3], delayed=dl, frame_out=fr)
    assert e.value.status == 1      # CFGMS_ERR_ARG
    for ctx, *_ in shards:
        ctx.close()


# ------------------------------------------------------------------ ragged per-stream vocabularies (W2 mask)
def test_ragged_stream_vocabularies_equal_truncated_heads(dev):
    """OpusLM-like shape: 9 streams of different vocabulary sizes on the padded uniform layout.  With the
    -inf tail mask installed by set_stream_vocab_sizes, every stream must sample exactly what the oracle
    samples from that stream's TRUNCATED head (a separate oracle run per distinct size on heads[:, :V_i]),
    i.e. padding + mask is the same computation as a ragged head."""
    wl = _custom(pairs=4, singles=2, d=128, S=9, V=512, T=20, mixed=True)
    wl.top_k[:] = 30
    sizes = [512, 200, 200, 384, 64, 512, 100, 37, 256]
    dw = DeviceWorkload(wl, dev)
    dw.ctx.set_stream_vocab_sizes(sizes)
    for t in (9, 12):
        dw.tokens.fill_(-1)
        dw.step(t)
        dw.check_no_device_error()
        got = dw.tokens.cpu().numpy()
        for Vi in sorted(set(sizes)):
            ref = oracle.step(wl.heads[:, :Vi].contiguous(), wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k,
                              wl.seed, wl.step(t), wl.req_id, wl.n_frames, wl.pad_token)
            for j, (c, i) in enumerate(ref.cells):
                if sizes[i] != Vi or ref.flags[j] & oracle.FLAG_INACTIVE:
                    continue
                assert got[c, i] < Vi
                if not ref.flags[j] & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
                    assert got[c, i] == ref.tok[j], (t, c, i, Vi)


@pytest.mark.parametrize("world", [1, 2, 3])
def test_device_side_token_exchange_between_stream_shards(dev, world):
    """W5 with the exchange done by the finalize kernel itself (cfgms_exchange_*): every 'rank' — here contexts of
    ONE process on ONE GPU, connected through their same-process block addresses, launched one after the other on
    one stream so that no kernel ever waits for a later one — stores its tokens into every rank's gather buffer and
    raises its flags; after the waits every rank holds the full [R][S] token matrix of the unsharded head.  Several
    steps (epochs, both halves of the double buffer), then a CUDA-graph replay of two more."""
    import paper_2607_02119_b200 as pkg
    from paper_2607_02119_b200 import dist_utils
    wl = _custom(pairs=5, singles=2, d=256, S=9, V=256, T=24, mixed=True)
    full = DeviceWorkload(wl, dev)
    R, S = wl.R, wl.S
    ranks = []
    for g in range(world):
        base, stride, s_local = dist_utils.stream_shard(g, world, S)
        heads = wl.heads[base::stride].contiguous().to(dev)
        embeds = wl.embeds[base::stride].contiguous().to(dev)
        ctx = pkg.Context(heads, embeds, max_rows=R, stream_base=base, stream_stride=stride, global_streams=S)
        handle, addr = ctx.exchange_create(world, g)
        assert len(handle) == 64 and addr
        ranks.append(dict(ctx=ctx, heads=heads, embeds=embeds, addr=addr,
                          tok=torch.full((R, s_local), -1, dtype=torch.int32, device=dev)))
    for rk in ranks:
        rk["ctx"].exchange_connect([x["addr"] for x in ranks])
        rk["all"] = rk["ctx"].exchange_tokens(R, S)

    def step_all(t, st):
        for rk in ranks:
            rk["ctx"].step(full.hidden(t), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, rk["tok"],
                           req_id=full.req_id, n_frames=full.n_frames)
        for rk in ranks:
            rk["ctx"].exchange_wait(R)

    for t in (0, 1, 4, 8, 9, 15, 23):
        full.step(t)
        step_all(t, wl.step(t).to(dev))
        torch.cuda.synchronize()
        for g, rk in enumerate(ranks):
            assert torch.equal(rk["all"], full.tokens), (t, g)
            rc, row = rk["ctx"].last_device_error()
            assert rc == 0
        check_tokens_against_oracle(wl, t, ranks[-1]["all"].cpu().numpy())     # the gathered matrix against the oracle itself
    # graph replay: the epochs live on the device
    sts = {t: wl.step(t).to(dev) for t in (10, 11)}
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        step_all(10, sts[10])
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    with torch.cuda.graph(g, stream=s):
        step_all(10, sts[10])
        step_all(11, sts[11])
    full.step(11)
    for _ in range(3):
        for rk in ranks:
            rk["all"].fill_(-5)
        g.replay()
        torch.cuda.synchronize()
        for rk in ranks:
            assert torch.equal(rk["all"], full.tokens)
    # the exchange needs the global stream count, and there is one per context
    with pytest.raises(pkg.CfgmsError):
        ranks[0]["ctx"].exchange_create(world, 0)
    # the binding hands the library exactly one block address per rank
    with pytest.raises(ValueError):
        ranks[0]["ctx"].exchange_connect([x["addr"] for x in ranks] + [ranks[0]["addr"]])
    with pytest.raises(ValueError):
        ranks[0]["ctx"].exchange_connect_ipc([b"\0" * 64] * (world + 1))
    # The request state advances on the PRIMARY stream's token: the rank that holds global stream 0 writes it (and
    # writes what the unsharded context writes); a rank without that stream is refused instead of silently leaving
    # step_next_out / n_frames_next_out / done_out untouched.
    st = wl.step(8).to(dev)
    mk = lambda: torch.full((R,), -9, dtype=torch.int32, device=dev)
    want = [mk(), mk(), mk()]
    full.ctx.step(full.hidden(8), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, full.tokens, req_id=full.req_id,
                  n_frames=full.n_frames, eos_token=3, step_next_out=want[0], n_frames_next_out=want[1], done_out=want[2])
    have = [mk(), mk(), mk()]
    ranks[0]["ctx"].step(full.hidden(8), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, ranks[0]["tok"],
                         req_id=full.req_id, n_frames=full.n_frames, eos_token=3, step_next_out=have[0],
                         n_frames_next_out=have[1], done_out=have[2])
    torch.cuda.synchronize()
    for a, b in zip(want, have):
        assert torch.equal(a, b) and bool((a.cpu().numpy()[wl.head_rows()] != -9).all())
    for rk in ranks[1:]:
        for kw in (dict(step_next_out=mk()), dict(n_frames_next_out=mk()), dict(done_out=mk())):
            with pytest.raises(pkg.CfgmsError) as e:
                rk["ctx"].step(full.hidden(8), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, rk["tok"],
                               req_id=full.req_id, n_frames=full.n_frames, **kw)
            assert e.value.status == 1      # CFGMS_ERR_ARG
    if world > 1:
        lone = pkg.Context(ranks[1]["heads"], ranks[1]["embeds"], max_rows=R, stream_base=1, stream_stride=world)
        with pytest.raises(pkg.CfgmsError):
            lone.exchange_create(world, 1)
        lone.close()
    for rk in ranks:
        rk["ctx"].close()


def test_exchange_wait_timeout_is_latched_and_the_context_survives(dev):
    """A peer that has not stepped yet: the wait gives up after its 2 s bound, latches CFGMS_ERR_TIMEOUT in the sticky
    error word and leaves the gathered tokens and its step count alone — no trap, the CUDA context stays usable — so
    the same step can be waited for again once the late peer has delivered."""
    import paper_2607_02119_b200 as pkg
    from paper_2607_02119_b200 import dist_utils
    wl = _custom(pairs=3, singles=2, d=128, S=4, V=128, T=16, mixed=True)
    full = DeviceWorkload(wl, dev)
    R, S = wl.R, wl.S
    ranks = []
    for g in range(2):
        base, stride, s_local = dist_utils.stream_shard(g, 2, S)
        heads = wl.heads[base::stride].contiguous().to(dev)
        embeds = wl.embeds[base::stride].contiguous().to(dev)
        ctx = pkg.Context(heads, embeds, max_rows=R, stream_base=base, stream_stride=stride, global_streams=S)
        _, addr = ctx.exchange_create(2, g)
        ranks.append(dict(ctx=ctx, heads=heads, embeds=embeds, addr=addr, tok=torch.full((R, s_local), -1, dtype=torch.int32, device=dev)))
    for rk in ranks:
        rk["ctx"].exchange_connect([x["addr"] for x in ranks])
    st = wl.step(6).to(dev)
    step = lambda rk: rk["ctx"].step(full.hidden(6), full.pair_map, full.w, full.temp, full.top_k, wl.seed, st, rk["tok"],
                                     req_id=full.req_id, n_frames=full.n_frames)
    step(ranks[0])
    ranks[0]["ctx"].exchange_wait(R)               # rank 1 has not stepped: 2 s, then the latch
    torch.cuda.synchronize()                       # a trap would surface here as a CUDA error
    assert ranks[0]["ctx"].last_device_error() == (7, 11)      # CFGMS_ERR_TIMEOUT, raised by the wait kernel
    assert ranks[0]["ctx"].last_device_error()[0] == 0
    step(ranks[1])                                 # the late peer delivers
    for rk in ranks:
        rk["ctx"].exchange_wait(R)
    full.step(6)
    torch.cuda.synchronize()
    for rk in ranks:
        assert rk["ctx"].last_device_error()[0] == 0
        assert torch.equal(rk["ctx"].exchange_tokens(R, S), full.tokens)
        rk["ctx"].close()
