"""GPU parity: the CUDA path, called through the C ABI, against the fp64 oracle on the same
seeded inputs.  Full BASELINE sizes, in the launch configuration bench.py times; at the large
configs the oracle computes a seeded sample of (request, stream) cells one by one."""
import numpy as np
import pytest
import torch

import oracle
import workloads
from parity_util import CLOSE_FRAC_MAX, DeviceWorkload, ParityStats, compare_step, sample_cells, valid_alternative

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    return torch.device("cuda:0")


def test_config1_tiny_all_steps_and_grid(dev):
    """BASELINE configs[0]: every token and every logit of all 24 steps, then the code grid."""
    wl = workloads.make_config(1)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    ref_delayed = np.full((wl.R, wl.T, wl.S), -1, dtype=np.int32)
    for t in range(wl.T):
        compare_step(dw, t, None, stats)
        oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                    wl.req_id, wl.n_frames, wl.pad_token, delayed=ref_delayed, hidden_is_f32=True)
    print("config1:", stats.summary())
    assert stats.n_pad == 2 * wl.S * (wl.S - 1)          # S(S-1)/2 head + tail PAD cells per request
    heads = wl.head_rows()
    gpu_delayed = dw.delayed.cpu().numpy()
    if stats.n_close_mismatch == 0:
        assert np.array_equal(gpu_delayed[heads], ref_delayed[heads])
    grid = dw.ctx.deinterleave(dw.delayed[torch.from_numpy(heads.astype(np.int64)).to(dev)].contiguous())
    torch.cuda.synchronize()
    assert grid.shape == (2, wl.T - wl.S + 1, wl.S)
    assert np.array_equal(grid.cpu().numpy(), oracle.deinterleave(gpu_delayed[heads]))
    assert (grid.cpu().numpy() != wl.pad_token).all()


def test_config2_mid_and_cfg_off_twin(dev):
    """BASELINE configs[1]: 64 pairs, d=2048, S=8, V=1024 + the CFG-off twin (64 cond rows)."""
    wl = workloads.make_config(2)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    for t in workloads.parity_steps(2, wl.T, wl.S):
        compare_step(dw, t, None, stats)
    print("config2:", stats.summary())
    stats.assert_close_fraction()
    off = workloads.cfg_off_twin(wl)
    dwo = DeviceWorkload(off, dev)
    so = ParityStats()
    for t in (0, 9, 130):
        compare_step(dwo, t, None, so)
    print("config2 cfg-off:", so.summary())
    # Without the w = 3 extrapolation the merged logits are ~3.6x narrower (std 1 instead of sqrt(9 + 4)), so the
    # top-50 perturbed scores lie ~3.6x denser and ties within 2e-2 are that much more frequent (observed 5.6 %).
    so.assert_close_fraction(frac=0.08)


def _full_step(cfg, T, S):
    """The parity step on which EVERY (request, stream) cell is checked (logits and tokens): the seeded
    mid-run step, where all streams are active.  The other parity steps check a seeded sample of cells."""
    steps = workloads.parity_steps(cfg, T, S)
    mid = [t for t in steps if S < t < T - S]
    return mid[0] if mid else steps[len(steps) // 2]


def test_config3_7b_head_heavy_tail(dev):
    wl = workloads.make_config(3)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    full = _full_step(3, wl.T, wl.S)
    for n, t in enumerate(workloads.parity_steps(3, wl.T, wl.S)):
        compare_step(dw, t, None if t == full else sample_cells(wl, 160, seed=30 + n), stats)   # full: all 1024 cells
    print("config3:", stats.summary())
    assert stats.n >= wl.n_req * wl.S
    stats.assert_close_fraction()


def test_config4_mixed_continuous_batch(dev):
    wl = workloads.make_config(4)
    dw = DeviceWorkload(wl, dev)
    # Two populations, counted apart: sampled cells of CFG pairs (the population SURVEY 8(c) simulated: 0.5-1.2 %
    # of them within 2e-2), and cells of unpaired or greedy requests, whose un-extrapolated logits are 2-5x
    # narrower (ties within 2e-2 that much denser; a greedy cell is close whenever the top-2 gap of M is: ~8 %
    # at V = 2048).
    pm, tk = wl.pair_map.numpy(), wl.top_k.numpy()
    is_cfg = lambda cells: np.asarray([pm[c] >= 0 and tk[c] != 1 for c, _ in cells])
    cfg_stats, rest_stats = ParityStats(), ParityStats()
    full = _full_step(4, wl.T, wl.S)
    for n, t in enumerate(workloads.parity_steps(4, wl.T, wl.S)):
        cells = sample_cells(wl, None if t == full else 320, seed=40 + n)      # full: all 2048 cells
        m = is_cfg(cells)
        compare_step(dw, t, cells[m], cfg_stats)
        compare_step(dw, t, cells[~m], rest_stats)
    print("config4 cfg pairs:", cfg_stats.summary())
    print("config4 unpaired / greedy:", rest_stats.summary())
    assert cfg_stats.n_pad + rest_stats.n_pad > 0          # step 0 has not-yet-started streams for low-offset rows
    assert cfg_stats.n + rest_stats.n >= wl.n_req * wl.S
    cfg_stats.assert_close_fraction()
    rest_stats.assert_close_fraction(frac=0.10)


def test_config5_large_batch(dev):
    wl = workloads.make_config(5)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    full = _full_step(5, wl.T, wl.S)
    for n, t in enumerate(workloads.parity_steps(5, wl.T, wl.S)):
        compare_step(dw, t, None if t == full else sample_cells(wl, 160, seed=50 + n), stats)   # full: all 8192 cells
    print("config5:", stats.summary())
    assert stats.n >= wl.n_req * wl.S
    stats.assert_close_fraction()
    info = dw.ctx.info()
    assert info["row_blocks"] == 4 and info["row_tile"] == 256


def test_config5_full_grid_deinterleave(dev):
    """[512][1024][16] int32 delayed buffer -> [512][1009][16] grid, bit-exact, in full."""
    wl = workloads.make_config(1)
    dw = DeviceWorkload(wl, dev)
    g = torch.Generator().manual_seed(5)
    delayed = torch.randint(0, 2049, (512, 1024, 16), generator=g, dtype=torch.int32)
    grid = dw.ctx.deinterleave(delayed.to(dev))
    torch.cuda.synchronize()
    assert grid.shape == (512, 1009, 16)
    assert np.array_equal(grid.cpu().numpy(), oracle.deinterleave(delayed.numpy()))


@pytest.mark.parametrize("n,T,S", [(3, 9, 9), (2, 40, 9), (5, 7, 1), (1, 300, 4), (4, 513, 16), (2, 258, 3), (0, 8, 4)])
def test_deinterleave_edge_shapes(dev, n, T, S):
    wl = workloads.make_config(1)
    dw = DeviceWorkload(wl, dev)
    g = torch.Generator().manual_seed(n * 1000 + T + S)
    delayed = torch.randint(-5, 5000, (n, T, S), generator=g, dtype=torch.int32)
    grid = dw.ctx.deinterleave(delayed.to(dev))
    torch.cuda.synchronize()
    assert grid.shape == (n, T - S + 1, S)
    if n:
        assert np.array_equal(grid.cpu().numpy(), oracle.deinterleave(delayed.numpy()))
        # host-buffer entry point gives the same grid
        assert np.array_equal(dw.ctx.deinterleave(delayed).numpy(), grid.cpu().numpy())


def _custom(pairs, singles, d, S, V, T=16, mixed=False, **kw):
    ov = dict(pairs=pairs, singles=singles, d=d, S=S, V=V, T=T, mixed=mixed, hidden_f32=False, heavy_tail=False)
    ov.update(kw)
    return workloads.make_config(2 if not mixed else 4, overrides=ov)


@pytest.mark.parametrize("case", [
    dict(pairs=0, singles=2, d=64, S=1, V=16),            # smallest: S = 1, one vocabulary tile, ragged
    dict(pairs=3, singles=0, d=72, S=3, V=100),           # K tail (d % 64 != 0), NT % 128 != 0
    dict(pairs=5, singles=6, d=256, S=9, V=520, mixed=True),   # OpusLM-like 9 streams, mixed slots
    dict(pairs=20, singles=8, d=128, S=4, V=12800),       # 400 vocabulary tiles: >2 tiles per CTA
    dict(pairs=100, singles=0, d=512, S=2, V=640),        # R = 200 -> one 224-row tile
    dict(pairs=150, singles=0, d=256, S=2, V=384),        # R = 300 -> two row blocks
    dict(pairs=3, singles=2, d=64, S=2, V=5000, top_k=700),    # 32 keys per thread; k > 256: no pruning bound
    dict(pairs=2, singles=2, d=64, S=1, V=9000, top_k=40),     # V > 8192: shared-memory sampler fallback
    dict(pairs=4, singles=0, d=64, S=2, V=1024, top_k=300),    # k > 256 with 4 keys per thread
    dict(pairs=4, singles=0, d=64, S=2, V=300, top_k=299),     # k = V - 1
])
def test_edge_shapes_full_oracle(dev, case):
    wl = _custom(**case)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    for t in (0, 1, wl.S, wl.T - 1):
        compare_step(dw, t, None, stats)
    print(case, stats.summary())


def test_candidate_overflow_chunks_and_full_scan_agree(dev):
    """The fused per-chunk top-4 candidate pass must stay exact when one 32-token chunk holds far more
    than four of the top-k (it is re-read in full), and must give the tokens of the full-scan sampler."""
    wl = _custom(pairs=6, singles=2, d=128, S=2, V=1024, top_k=40)
    wl.heads[0, 64:90] *= 5.0           # 26 hot tokens inside chunk 2 of stream 0 (and chunk 2 only partly)
    wl.heads[1, 500:520] *= 4.0         # straddles chunks 15 and 16 of stream 1
    stats = ParityStats()
    dw = DeviceWorkload(wl, dev)
    for t in (3, 8, 12):
        compare_step(dw, t, None, stats)
    print("overflow:", stats.summary())
    full = DeviceWorkload(wl, dev, no_candidates=True)
    for t in (3, 8):
        dw.step(t)
        full.step(t)
        torch.cuda.synchronize()
        assert torch.equal(dw.tokens, full.tokens)
    # the full-scan sampler on its own is also exact against the oracle
    s2 = ParityStats()
    compare_step(full, 5, None, s2)
    # every per-row mode of the candidate path against the full-scan path at a BASELINE shape
    wl2 = _custom(pairs=24, singles=16, d=256, S=4, V=2048, mixed=True)
    heads = wl2.head_rows()
    modes = [0, 1, 20, 50, 256, 257, 2047, 2048, 5000, -1]
    for q, r in enumerate(heads):
        wl2.top_k[r] = modes[q % len(modes)]
    a, b = DeviceWorkload(wl2, dev), DeviceWorkload(wl2, dev, no_candidates=True)
    s3 = ParityStats()
    compare_step(a, 9, None, s3)
    for t in (4, 9):
        a.step(t)
        b.step(t)
        torch.cuda.synchronize()
        assert torch.equal(a.tokens, b.tokens)


def test_row_tile_override_many_row_blocks(dev):
    """Force 64-row accumulator tiles: 4 row blocks x 10 vocabulary tiles through the same kernel."""
    wl = _custom(pairs=100, singles=8, d=192, S=2, V=640, mixed=True)
    dw = DeviceWorkload(wl, dev, row_tile=64)
    stats = ParityStats()
    for t in (0, 5):
        compare_step(dw, t, None, stats)
    assert dw.ctx.info()["row_blocks"] == 4
    # tile shape must not change any token (determinism across tilings)
    dw2 = DeviceWorkload(wl, dev, row_tile=0)
    dw.step(7)
    dw2.step(7)
    torch.cuda.synchronize()
    assert torch.equal(dw.tokens, dw2.tokens)


def test_odd_row_count_and_single_row(dev):
    wl = _custom(pairs=2, singles=2, d=128, S=4, V=256)
    # drop the last row: R = 5, last slot holds one unpaired row
    import dataclasses
    cut = lambda a: None if a is None else a[:5].clone()
    wl5 = dataclasses.replace(wl, R=5, n_req=3, hidden_pool=wl.hidden_pool[:, :5].clone(), pair_map=cut(wl.pair_map),
                              w=cut(wl.w), temp=cut(wl.temp), top_k=cut(wl.top_k), req_id=cut(wl.req_id),
                              n_frames=cut(wl.n_frames), offset=cut(wl.offset))
    stats = ParityStats()
    compare_step(DeviceWorkload(wl5, dev), 6, None, stats)
    one = lambda a: None if a is None else a[4:5].clone()
    wl1 = dataclasses.replace(wl, R=1, n_req=1, hidden_pool=wl.hidden_pool[:, 4:5].clone(), pair_map=one(wl.pair_map),
                              w=one(wl.w), temp=one(wl.temp), top_k=one(wl.top_k), req_id=one(wl.req_id),
                              n_frames=one(wl.n_frames), offset=one(wl.offset))
    s1 = ParityStats()
    got1 = compare_step(DeviceWorkload(wl1, dev), 6, None, s1)
    # a request alone gives the same tokens as inside the batch (counter-based noise)
    dw5 = DeviceWorkload(wl5, dev)
    dw5.step(6)
    torch.cuda.synchronize()
    assert np.array_equal(dw5.tokens.cpu().numpy()[4], got1[0])


def test_sampler_parameter_edges(dev):
    """top_k <= 0, top_k >= V, top_k = 1, temp = 0, w = 0, w = 1, per-row mixes."""
    wl = _custom(pairs=8, singles=0, d=128, S=4, V=256)
    heads = wl.head_rows()
    tk = [0, -3, 256, 1000, 1, 50, 2, 255]
    tp = [1.0, 0.7, 1.3, 0.9, 0.8, 0.0, 1e-4, 1.0]
    ww = [3.0, 0.0, 1.0, 2.5, 3.0, 3.0, -1.0, 7.5]
    for q, r in enumerate(heads):
        wl.top_k[r] = tk[q]
        wl.temp[r] = tp[q]
        wl.w[r] = ww[q]
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    for t in (3, 9):
        got = compare_step(dw, t, None, stats)
    print("sampler edges:", stats.summary())
    # greedy rows equal the argmax of the merged logits the GPU itself reports
    logits = torch.zeros((wl.R, wl.S, wl.V), dtype=torch.float32, device=dev)
    dw.step(9, logits_out=logits)
    torch.cuda.synchronize()
    am = logits.argmax(dim=-1).cpu().numpy()
    for q in (4, 5):
        assert np.array_equal(dw.tokens.cpu().numpy()[heads[q]], am[heads[q]])


def test_w1_equals_noncfg_and_tokens_independent_of_placement(dev):
    wl = _custom(pairs=6, singles=0, d=256, S=4, V=512)
    wl.w[:] = 1.0
    off = workloads.cfg_off_twin(wl)
    a, b = DeviceWorkload(wl, dev), DeviceWorkload(off, dev)
    for t in (4, 11):
        a.step(t)
        b.step(t)
        torch.cuda.synchronize()
        assert np.array_equal(a.tokens.cpu().numpy()[wl.head_rows()], b.tokens.cpu().numpy())


def test_ring_buffer_depth_S(dev):
    wl = workloads.make_config(1)
    ring = DeviceWorkload(wl, dev, T_cap=wl.S)
    full = DeviceWorkload(wl, dev)
    for t in range(11):
        ring.step(t)
        full.step(t)
    torch.cuda.synchronize()
    r, f = ring.delayed.cpu().numpy(), full.delayed.cpu().numpy()
    for t in range(7, 11):
        assert np.array_equal(r[:, t % wl.S], f[:, t])


def test_step_host_matches_device_path(dev):
    wl = _custom(pairs=10, singles=4, d=256, S=4, V=384, mixed=True)
    dw = DeviceWorkload(wl, dev)
    dw.step(5)
    torch.cuda.synchronize()
    tok_host = torch.full((wl.R, wl.S), -1, dtype=torch.int32).pin_memory()
    dw.ctx.step_host(wl.hidden(5).pin_memory(), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(5), tok_host,
                     req_id=wl.req_id, n_frames=wl.n_frames)
    assert torch.equal(tok_host, dw.tokens.cpu())
    inf = dw.ctx.info()
    assert inf["h2d_bytes_last_step"] >= wl.R * wl.d * 2 and inf["d2h_bytes_last_step"] == wl.R * wl.S * 4


def test_errors_are_reported_not_fatal(dev):
    import paper_2607_02119_b200 as pkg
    wl = _custom(pairs=4, singles=0, d=128, S=2, V=128)
    dw = DeviceWorkload(wl, dev)
    bad = wl.pair_map.clone()
    bad[0], bad[1] = -1, 0            # row 1 claims row 0, row 0 does not claim back
    dw.pair_map = bad.to(dev)
    dw.step(3)
    torch.cuda.synchronize()
    rc, row = dw.ctx.last_device_error()
    assert rc == 3 and row == 0       # CFGMS_ERR_LAYOUT at the slot's even row
    assert dw.ctx.last_device_error()[0] == 0          # sticky word cleared
    # host-side validation
    for bits in (256, 512):           # the measurement probes' flag bits: only the probe build of the library knows them
        with pytest.raises(pkg.CfgmsError) as e:
            pkg.Context(dw.heads, dw.embeds, max_rows=4, probe=bits)
        assert e.value.status == 1
    small = pkg.Context(dw.heads, dw.embeds, max_rows=4)
    with pytest.raises(pkg.CfgmsError) as e:
        small.step(dw.hidden(0), dw.pair_map, dw.w, dw.temp, dw.top_k, 0, wl.step(0).to(dev), dw.tokens)
    assert e.value.status == 2        # CFGMS_ERR_SHAPE: R > max_rows
    with pytest.raises(pkg.CfgmsError):
        pkg.Context(dw.heads[:, :, :12].contiguous(), dw.embeds[:, :12].contiguous())    # d % 8 != 0
    # the context still works after errors
    dw.pair_map = wl.pair_map.to(dev)
    compare_step(dw, 3, None, ParityStats())


def test_overlapped_finalize_equals_serial_finalize(dev):
    """K2 launched as a programmatic dependent of K1 (consuming finished (stream, row block) groups
    through the ready counters) must sample exactly what the strictly
    serial launch samples; many consecutive steps also exercise the counter re-arm, a multi-wave
    GEMM (row_tile 64 -> several row blocks) and CUDA-graph replay of the programmatic edge."""
    wl = workloads.make_config(2)
    ov = DeviceWorkload(wl, dev, force_overlap=True)
    ov64 = DeviceWorkload(wl, dev, row_tile=64, force_overlap=True)
    ser = DeviceWorkload(wl, dev, no_overlap=True)
    for t in (0, 3, 8, 9, 10, 100, 250, 255):
        for dw in (ov, ov64, ser):
            dw.step(t)
        torch.cuda.synchronize()
        assert torch.equal(ov.tokens, ser.tokens) and torch.equal(ov64.tokens, ser.tokens)
    assert torch.equal(ov.delayed, ser.delayed)
    assert ov.ctx.info()["overlap"] == 1 and ser.ctx.info()["overlap"] == 0
    assert ov.ctx.overlap_stats() >= 0 and ser.ctx.overlap_stats() == 0
    # graph replay of the programmatic edge: the captured pair of steps, replayed, equals eager
    steps = {t: wl.step(t).to(dev) for t in (20, 21)}
    run = lambda t: ov.ctx.step(ov.hidden(t), ov.pair_map, ov.w, ov.temp, ov.top_k, wl.seed, steps[t], ov.tokens,
                                req_id=ov.req_id, n_frames=ov.n_frames, delayed=ov.delayed)
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        run(20)
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    with torch.cuda.graph(g, stream=s):
        run(20)
        run(21)
    ser.step(21)
    torch.cuda.synchronize()
    for _ in range(3):
        ov.tokens.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(ov.tokens, ser.tokens)
    ov.check_no_device_error()


def test_finalize_really_runs_beside_the_large_gemm(dev):
    """Config 5 in the default policy: the finalize kernel must be RESIDENT beside the head GEMM, i.e. a good share of its
    cells reach their readiness check before the GEMM has finished their group.  (Regression: a head GEMM that asks for
    less shared memory lets the driver pick a smaller carve-out, the finalize CTAs no longer fit, everything still
    computes the same tokens — and the overlap silently turns into a serial launch.)"""
    wl = workloads.make_config(5)
    dw = DeviceWorkload(wl, dev)
    for t in (16, 17, 18):
        dw.step(t)
    torch.cuda.synchronize()
    assert dw.ctx.info()["overlap"] == 1
    waited = dw.ctx.overlap_stats()
    assert waited >= 3 * wl.n_req * wl.S // 4, f"only {waited} of {3 * wl.n_req * wl.S} cells met a running GEMM"
    dw.check_no_device_error()


def test_overlap_counters_survive_steps_whose_cells_are_mostly_pad(dev):
    """Regression: at tau = 0 only stream 0 samples; if PAD cells did not wait for their group the
    finalize grid could finish (and re-arm the ready counters) while the GEMM was still signalling,
    and the NEXT step would read unfinished tiles.  Multi-wave overlapped GEMM (8 row blocks x 64
    vocabulary tiles), PAD-heavy and full steps alternating, against the strictly serial launch."""
    wl = _custom(pairs=256, singles=0, d=512, S=8, V=1024, T=64)
    ov = DeviceWorkload(wl, dev, row_tile=64, force_overlap=True)
    ser = DeviceWorkload(wl, dev, no_overlap=True)
    for rep in range(12):
        for t in (0, 9, 1, 30, wl.T - 1, 12):
            ov.step(t)
            ser.step(t)
            torch.cuda.synchronize()
            assert torch.equal(ov.tokens, ser.tokens), (rep, t)
    assert ov.ctx.info()["overlap"] == 1
    ov.check_no_device_error()


@pytest.mark.parametrize("cfg,n_cells", [(5, 96), (4, 96), (3, 64), (2, 256)])
def test_bench_launch_configuration_graph_replay(dev, cfg, n_cells):
    """The launch configuration bench.py times: default policy (config 5: lean GEMM + dependent finalize
    beside it; configs 2-4: full-register GEMM, serial finalize), no debug tap, consecutive steps
    captured in ONE CUDA graph and replayed.  Tokens of every captured step are read back from the
    delayed buffer and compared with the oracle on a seeded sample of cells."""
    wl = workloads.make_config(cfg)
    dw = DeviceWorkload(wl, dev)
    steps = [0, wl.S - 1, wl.S + 2, 40, 41, 42]
    st = {t: wl.step(t).to(dev) for t in steps}
    run = lambda t: dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, st[t], dw.tokens,
                                req_id=dw.req_id, n_frames=dw.n_frames, delayed=dw.delayed)
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        run(steps[0])
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    with torch.cuda.graph(g, stream=s):
        for t in steps:
            run(t)
    dw.delayed.fill_(-1)
    g.replay()
    g.replay()
    dw.check_no_device_error()
    assert dw.ctx.info()["overlap"] == (1 if cfg == 5 else 0)
    delayed = dw.delayed.cpu().numpy()
    n_close = n_mismatch = n_sampled = 0
    for n, t in enumerate(steps):
        cells = sample_cells(wl, n_cells, seed=900 + n)
        ref = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                          wl.req_id, wl.n_frames, wl.pad_token, cells=cells, hidden_is_f32=wl.hidden_f32)
        tau = wl.step(t).numpy()
        for j, (c, i) in enumerate(ref.cells):
            got = delayed[c, int(tau[c]) % dw.T_cap, i]
            if ref.flags[j] & oracle.FLAG_INACTIVE:
                assert got == wl.pad_token
                continue
            n_sampled += 1
            if ref.flags[j] & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
                n_close += 1
                if got != ref.tok[j]:
                    n_mismatch += 1
                    assert valid_alternative(wl, t, c, i, int(got)), (t, c, i, got, ref.tok[j], ref.margin[j])
            else:
                assert got == ref.tok[j], (t, c, i, got, ref.tok[j], ref.margin[j])
    print(f"config{cfg} graph replay: {n_sampled} sampled cells, close ties {n_close}, of which differ {n_mismatch}")
    # config 4 mixes in unpaired and greedy requests, whose un-extrapolated logits tie within 2e-2 several times more often
    # (the two populations are counted apart, with this same 0.10 bound, in test_config4_mixed_continuous_batch)
    assert n_mismatch <= n_close <= (0.10 if cfg == 4 else CLOSE_FRAC_MAX) * n_sampled + 2
