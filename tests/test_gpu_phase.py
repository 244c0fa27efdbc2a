"""GPU parity of the per-request phase state machine (widening W6; DESIGN.md readings
C28-C32) against the oracle, through the C ABI: a mixed batch is driven through text -> transition ->
audio -> drain -> done with the state living on the device (phase, position, step, frame count fed back
from one step's outputs to the next), and every step's tokens, modality inference, logits and state are
compared with oracle.step_phase / oracle.phase_advance."""
import numpy as np
import pytest
import torch

import oracle
import workloads
from oracle import F_UNSET, PHASE_AUDIO, PHASE_DONE, PHASE_TEXT, PHASE_TRANSITION
from parity_util import LOGIT_TOL, DeviceWorkload

pytestmark = pytest.mark.gpu


def _custom(pairs, singles, d, S, V, T=16, mixed=True, **kw):
    ov = dict(pairs=pairs, singles=singles, d=d, S=S, V=V, T=T, mixed=mixed, hidden_f32=False, heavy_tail=False)
    ov.update(kw)
    return workloads.make_config(4 if mixed else 2, overrides=ov)


@pytest.mark.parametrize("case", [
    dict(V=512, V_text=192, no_candidates=False, bridge=[500, 3, 260], eos=300),     # candidate sampler (V % 32 == 0)
    dict(V=512, V_text=192, no_candidates=True, bridge=[7], eos=300),                # block-per-cell sampler
    dict(V=200, V_text=70, no_candidates=False, bridge=[], eos=150),                 # V % 32 != 0: any region; no bridging
    dict(V=512, V_text=192, no_candidates=False, bridge=[9, 400], eos=300, d=512),   # deep enough for the split-K head GEMM
])
def test_mixed_batch_through_all_phases(case):
    dev = torch.device("cuda:0")
    V, V_text, bridge, EOS = case["V"], case["V_text"], case["bridge"], case["eos"]
    wl = _custom(pairs=6, singles=4, d=case.get("d", 256), S=4, V=V, T=64)
    R, S = wl.R, wl.S
    heads = wl.head_rows()
    pm = wl.pair_map.numpy()
    dw = DeviceWorkload(wl, dev, T_cap=16, no_candidates=case["no_candidates"])
    dw.ctx.set_phase_table(V_text, bridge)
    # the end-of-audio id and the audio region of stream 0 get a push so that requests change phase within the window
    bias = np.zeros((S, V), dtype=np.float32)
    bias[0, EOS] = 2.0
    bias[0, V_text:] += 0.5
    dw.ctx.set_logit_bias(torch.from_numpy(bias).to(dev))
    rng = np.random.default_rng(5)
    # requests start in different phases and at different global steps (a continuous batch)
    o_phase = np.zeros(R, dtype=np.int32)
    o_pos = np.zeros(R, dtype=np.int32)
    o_gstep = np.zeros(R, dtype=np.int32)
    o_F = np.full(R, F_UNSET, dtype=np.int32)
    for q, c in enumerate(heads):
        o_gstep[c] = int(rng.integers(0, 50))
        if q % 5 == 1:
            o_phase[c], o_pos[c] = PHASE_AUDIO, int(rng.integers(0, 6))
        elif q % 5 == 2 and bridge:
            o_phase[c], o_pos[c] = PHASE_TRANSITION, len(bridge) - 1
    mk = lambda a: [torch.from_numpy(a.copy()).to(dev), torch.zeros(R, dtype=torch.int32, device=dev)]
    g_phase, g_pos, g_gstep, g_F = mk(o_phase), mk(o_pos), mk(o_gstep), mk(o_F)
    done = torch.zeros(R, dtype=torch.int32, device=dev)
    modality = torch.zeros(R, dtype=torch.int32, device=dev)
    seen = set()
    n_close = n_mod_close = n_cells = 0
    for t in range(40):
        a, b = t & 1, (t + 1) & 1
        logits = torch.zeros((R, S, V), dtype=torch.float32, device=dev)
        dw.tokens.fill_(-7)
        before = dw.delayed.clone()
        dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, g_gstep[a], dw.tokens, req_id=dw.req_id,
                    n_frames=g_F[a], delayed=dw.delayed, logits_out=logits, eos_token=EOS, step_next_out=g_gstep[b],
                    n_frames_next_out=g_F[b], done_out=done, phase=g_phase[a], phase_pos=g_pos[a],
                    phase_next_out=g_phase[b], phase_pos_next_out=g_pos[b], modality_out=modality)
        dw.check_no_device_error()
        ref = oracle.step_phase(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, o_gstep,
                                o_phase, o_pos, V_text, bridge, req_id=wl.req_id, n_frames=o_F, pad_token=wl.pad_token,
                                want_merged=True, logit_bias=bias.astype(np.float64))
        got, gl = dw.tokens.cpu().numpy(), logits.cpu().numpy().astype(np.float64)
        g_mod, g_done = modality.cpu().numpy(), done.cpu().numpy()
        dl, dl0 = dw.delayed.cpu().numpy(), before.cpu().numpy()
        tok0, mod = {}, {}
        for j, (c, i) in enumerate(ref.cells):
            n_cells += 1
            fl = int(ref.flags[j])
            seen.add(int(o_phase[c]))
            if pm[c] >= 0:
                assert got[pm[c], i] == got[c, i]                      # companion receives the token in every phase
            if fl & (oracle.FLAG_INACTIVE | oracle.FLAG_FORCED):
                assert got[c, i] == ref.tok[j], (t, c, i, o_phase[c], got[c, i], ref.tok[j])      # pad / bridging token: exact
            else:
                m = ref.merged[j]
                # TEXT phase: the tap must show the conditional row's logits alone (merge bypassed)
                assert np.max(np.abs(gl[c, i] - m)) <= LOGIT_TOL, (t, c, i, o_phase[c])
                lo, hi = (0, V_text) if o_phase[c] == PHASE_TEXT else ((V_text, V) if i == 0 else (0, V))
                assert lo <= got[c, i] < hi, (t, c, i, got[c, i])      # dynamic vocabulary masking: never outside the region
                if fl & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
                    n_close += 1
                else:
                    assert got[c, i] == ref.tok[j], (t, c, i, o_phase[c], got[c, i], ref.tok[j], ref.margin[j])
            if i == 0:
                tok0[int(c)] = int(got[c, i])
                want_mod = int(ref.modality[j])
                if o_phase[c] == PHASE_TEXT:
                    m = ref.merged[j]
                    if abs(m[:V_text].max() - m[V_text:].max()) <= LOGIT_TOL:      # the two regions tie within the logit tolerance
                        n_mod_close += 1
                    else:
                        assert g_mod[c] == want_mod, (t, c, g_mod[c], want_mod)
                else:
                    assert g_mod[c] == 0
                mod[int(c)] = int(g_mod[c])
            # the delayed buffer takes audio-phase tokens only, at the audio-local slot
            if o_phase[c] == PHASE_AUDIO:
                assert dl[c, o_pos[c] % dw.T_cap, i] == got[c, i]
            else:
                assert np.array_equal(dl[c, :, i], dl0[c, :, i])
        # state: the oracle's transition function applied to what the GPU emitted must give the GPU's next state
        np_phase, np_pos, np_gstep, np_F = (x[b].cpu().numpy() for x in (g_phase, g_pos, g_gstep, g_F))
        for c in heads:
            ph, pos, F, d = oracle.phase_advance(int(o_phase[c]), int(o_pos[c]), int(o_F[c]), tok0[int(c)], bool(mod[int(c)]),
                                                 len(bridge), EOS, S)
            assert (np_phase[c], np_pos[c], np_F[c], bool(g_done[c])) == (ph, pos, F, d), (t, c, o_phase[c], o_pos[c])
            assert np_gstep[c] == o_gstep[c] + 1
            o_phase[c], o_pos[c], o_F[c], o_gstep[c] = ph, pos, F, o_gstep[c] + 1
    print(f"phase machine {case}: {n_cells} cells, {n_close} close, {n_mod_close} modality ties; phases seen {sorted(seen)}; "
          f"final phases {sorted(int(o_phase[c]) for c in heads)}")
    assert {PHASE_TEXT, PHASE_AUDIO, PHASE_DONE} <= seen | {int(o_phase[c]) for c in heads}
    if bridge:
        assert PHASE_TRANSITION in seen
    assert n_close <= 0.1 * n_cells and n_mod_close <= 3


def test_phase_arguments_are_validated():
    import paper_2607_02119_b200 as pkg
    dev = torch.device("cuda:0")
    wl = _custom(pairs=2, singles=0, d=64, S=2, V=128, mixed=False)
    dw = DeviceWorkload(wl, dev)
    ph = torch.zeros(wl.R, dtype=torch.int32, device=dev)
    args = (dw.hidden(0), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, wl.step(0).to(dev), dw.tokens)
    with pytest.raises(pkg.CfgmsError) as e:
        dw.ctx.step(*args, phase=ph)                                   # phase without phase_pos
    assert e.value.status == 1
    with pytest.raises(pkg.CfgmsError):
        dw.ctx.step(*args, phase_pos=ph)                               # phase_pos without phase
    with pytest.raises(pkg.CfgmsError):
        dw.ctx.step(*args, phase=ph, phase_pos=ph, force_token=torch.full((wl.R, wl.S), -1, dtype=torch.int32, device=dev))
    with pytest.raises(pkg.CfgmsError) as e:
        dw.ctx.set_phase_table(50, [1])                                # candidate path: regions are whole 32-token chunks
    assert e.value.status == 2
    with pytest.raises(pkg.CfgmsError):
        dw.ctx.set_phase_table(64, list(range(17)))                    # at most 16 bridging tokens
    dw.ctx.set_phase_table(64, [1, 2])
    # an all-audio phase vector with phase_pos = step and an empty text region is the plain path
    dw.ctx.set_phase_table(0, [])
    dw.step(5)
    torch.cuda.synchronize()
    plain = dw.tokens.clone()
    dw.tokens.fill_(-1)
    st = wl.step(5).to(dev)
    dw.ctx.step(dw.hidden(5), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, st, dw.tokens, req_id=dw.req_id,
                n_frames=dw.n_frames, delayed=dw.delayed, phase=torch.full((wl.R,), 2, dtype=torch.int32, device=dev), phase_pos=st)
    torch.cuda.synchronize()
    assert torch.equal(plain, dw.tokens)


@pytest.mark.parametrize("no_candidates", [False, True])
def test_text_phase_with_an_empty_text_region_moves_on(no_candidates):
    """`phase` passed without a phase table (V_text = 0, no bridging tokens): a TEXT-phase request has nothing to
    sample, pads — and its unmasked argmax necessarily lies in the audio region, so the modality inference says
    "audio" and the request enters the audio phase at the next step, exactly as oracle.step_phase /
    oracle.phase_advance say (it must not sit in TEXT forever)."""
    dev = torch.device("cuda:0")
    wl = _custom(pairs=3, singles=2, d=128, S=3, V=160 if no_candidates else 256, T=16)
    R, S = wl.R, wl.S
    dw = DeviceWorkload(wl, dev, no_candidates=no_candidates)
    heads = wl.head_rows()
    o_phase = np.full(R, PHASE_TEXT, dtype=np.int32)
    o_pos = np.zeros(R, dtype=np.int32)
    o_gstep = np.arange(R, dtype=np.int32)
    o_F = np.full(R, F_UNSET, dtype=np.int32)
    cu = lambda a: torch.from_numpy(a.copy()).to(dev)
    out = {k: torch.full((R,), -9, dtype=torch.int32, device=dev) for k in ("phase", "pos", "gstep", "F", "done", "mod")}
    dw.tokens.fill_(-7)
    dw.ctx.step(dw.hidden(0), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, cu(o_gstep), dw.tokens, req_id=dw.req_id,
                n_frames=cu(o_F), delayed=dw.delayed, eos_token=5, step_next_out=out["gstep"], n_frames_next_out=out["F"],
                done_out=out["done"], phase=cu(o_phase), phase_pos=cu(o_pos), phase_next_out=out["phase"],
                phase_pos_next_out=out["pos"], modality_out=out["mod"])
    dw.check_no_device_error()
    ref = oracle.step_phase(wl.heads, wl.embeds, wl.hidden(0), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, o_gstep,
                            o_phase, o_pos, 0, [], req_id=wl.req_id, n_frames=o_F, pad_token=wl.pad_token)
    got = dw.tokens.cpu().numpy()
    for j, (c, i) in enumerate(ref.cells):
        assert ref.tok[j] == wl.pad_token and got[c, i] == wl.pad_token
        if i == 0:
            assert ref.modality[j] == 1
    res = {k: v.cpu().numpy() for k, v in out.items()}
    for c in heads:
        ph, pos, F, d = oracle.phase_advance(PHASE_TEXT, 0, F_UNSET, wl.pad_token, True, 0, 5, S)
        assert ph == PHASE_AUDIO
        assert (res["mod"][c], res["phase"][c], res["pos"][c], res["F"][c], bool(res["done"][c])) == (1, ph, pos, F, d), c
        assert res["gstep"][c] == o_gstep[c] + 1


def test_step_host_stages_the_phase_inputs():
    """cfgms_step_host takes phase / phase_pos as HOST arrays like its other inputs (they travel in the one packed
    parameter copy); tokens and the device-resident next state equal cfgms_step's on a batch that holds every phase."""
    dev = torch.device("cuda:0")
    V, V_text, bridge, EOS = 512, 192, [500, 3], 300
    wl = _custom(pairs=6, singles=4, d=256, S=4, V=V, T=64)
    R, S = wl.R, wl.S
    dw = DeviceWorkload(wl, dev, T_cap=16)
    dw.ctx.set_phase_table(V_text, bridge)
    phase = torch.zeros(R, dtype=torch.int32)
    pos = torch.zeros(R, dtype=torch.int32)
    for q, c in enumerate(wl.head_rows()):
        phase[c] = q % 4
        pos[c] = 1 if q % 4 == PHASE_TRANSITION else (q if q % 4 == PHASE_AUDIO else 0)
    gstep = torch.arange(R, dtype=torch.int32) + 3
    names = ("step_next_out", "n_frames_next_out", "done_out", "phase_next_out", "phase_pos_next_out", "modality_out")
    mk = lambda: {k: torch.full((R,), -9, dtype=torch.int32, device=dev) for k in names}
    want, have = mk(), mk()
    dw.tokens.fill_(-7)
    dw.ctx.step(dw.hidden(2), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, gstep.to(dev), dw.tokens, req_id=dw.req_id,
                n_frames=dw.n_frames, eos_token=EOS, phase=phase.to(dev), phase_pos=pos.to(dev), **want)
    dw.check_no_device_error()
    tok_host = torch.full((R, S), -1, dtype=torch.int32).pin_memory()
    dw.ctx.step_host(wl.hidden(2).pin_memory(), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, gstep, tok_host,
                     req_id=wl.req_id, n_frames=wl.n_frames, eos_token=EOS, phase=phase, phase_pos=pos, **have)
    dw.check_no_device_error()
    assert torch.equal(tok_host, dw.tokens.cpu())
    assert len({int(x) for x in phase.numpy()[wl.head_rows()]}) == 4
    for k in names:
        assert torch.equal(want[k], have[k]), k
        assert bool((want[k].cpu().numpy()[wl.head_rows()] != -9).all()), k
    n_arrays = 5 + 2 + (wl.req_id is not None) + (wl.n_frames is not None)      # the plain path's [R] inputs + phase, phase_pos
    assert dw.ctx.info()["h2d_bytes_last_step"] == R * wl.d * 2 + n_arrays * R * 4
