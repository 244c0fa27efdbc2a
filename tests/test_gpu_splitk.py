"""Split-K head GEMM (one-wave shapes: clusters of four CTAs, two cta_group::2 pairs each streaming half of K,
partial sums exchanged over distributed shared memory — csrc/head_gemm.cuh).
Parity with the fp64 oracle on every cell (logits through the tap, tokens), on the shapes the split-K
epilogue distinguishes, and bit-equality of the sampled tokens with the plain (row-split) GEMM."""
import numpy as np
import pytest
import torch

import workloads
from parity_util import DeviceWorkload, ParityStats, compare_step

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    return torch.device("cuda:0")


def _custom(pairs, singles, d, S, V, T=16, mixed=False, **kw):
    ov = dict(pairs=pairs, singles=singles, d=d, S=S, V=V, T=T, mixed=mixed, hidden_f32=False, heavy_tail=False)
    ov.update(kw)
    return workloads.make_config(2 if not mixed else 4, overrides=ov)


CASES = [
    dict(pairs=64, singles=0, d=2048, S=2, V=1024),              # 128 rows: both column halves owned, CFG pairs only
    dict(pairs=0, singles=64, d=1024, S=2, V=512),               # <= 64 rows, all unpaired: even / odd passes on different warps
    dict(pairs=20, singles=0, d=512, S=3, V=384),                # <= 64 rows, pairs only: the odd-row warps idle
    dict(pairs=9, singles=14, d=768, S=2, V=640, mixed=True),    # <= 64 rows, pairs and unpaired slots interleaved
    dict(pairs=30, singles=38, d=512, S=2, V=256, mixed=True),   # 98 rows: ragged second column half
    dict(pairs=100, singles=0, d=512, S=2, V=640),               # 200 rows: two 128-row blocks, ten clusters
    dict(pairs=40, singles=0, d=584, S=1, V=896),                # K tail (d % 64 != 0) split unevenly; odd number of vocabulary tiles
    dict(pairs=3, singles=2, d=512, S=5, V=160, mixed=True),     # chunks that straddle nothing: NT = 800, last tile ragged
]


@pytest.mark.parametrize("case", CASES)
def test_split_k_full_oracle_parity(dev, case):
    wl = _custom(**case)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    for t in (0, 1, wl.S, wl.T - 1):
        compare_step(dw, t, None, stats)
    assert dw.ctx.info()["split_k"] == 2
    print(case, stats.summary())


@pytest.mark.parametrize("case", CASES[:6])
def test_split_k_tokens_equal_plain_gemm(dev, case):
    """Same tokens as the GEMM that splits the rows instead of K, except where the two summation orders move a
    logit across a tie (counted: the fp32 partial sums differ in the last bits)."""
    wl = _custom(**case)
    a = DeviceWorkload(wl, dev)
    b = DeviceWorkload(wl, dev, no_split_k=True)
    diff = total = 0
    for t in (0, 2, wl.S, wl.S + 3, wl.T - 1):
        la = torch.zeros((wl.R, wl.S, wl.V), dtype=torch.float32, device=dev)
        lb = torch.zeros_like(la)
        a.step(t, logits_out=la)
        b.step(t, logits_out=lb)
        torch.cuda.synchronize()
        rows = torch.as_tensor(wl.head_rows(), device=dev, dtype=torch.long)
        assert float((la[rows] - lb[rows]).abs().max()) <= 1e-3
        diff += int((a.tokens != b.tokens).sum())
        total += a.tokens.numel()
    assert a.ctx.info()["split_k"] == 2 and b.ctx.info()["split_k"] == 1
    assert diff <= max(2, total // 200), f"{diff} of {total} tokens differ between the split-K and the plain GEMM"


def test_split_k_in_a_graph_and_after_other_shapes(dev):
    """One context, batches of changing size (128 -> 40 -> 128 rows: the epilogue's column ownership changes with R),
    then a captured graph of consecutive split-K steps replayed twice: tokens equal the eager run."""
    wl = workloads.make_config(2)
    dw = DeviceWorkload(wl, dev)
    stats = ParityStats()
    compare_step(dw, 9, None, stats)
    small = _custom(pairs=12, singles=16, d=wl.d, S=wl.S, V=wl.V, mixed=True)
    small.heads, small.embeds = wl.heads, wl.embeds           # same head, smaller batch, same context
    ds = DeviceWorkload(small, dev)
    ds.ctx = dw.ctx
    compare_step(ds, 9, None, stats)
    compare_step(dw, 10, None, stats)
    steps = {t: wl.step(t).to(dev) for t in (20, 21, 22)}
    run = lambda t: dw.ctx.step(dw.hidden(t), dw.pair_map, dw.w, dw.temp, dw.top_k, wl.seed, steps[t], dw.tokens,
                                req_id=dw.req_id, n_frames=dw.n_frames, delayed=dw.delayed)
    eager = []
    for t in (20, 21, 22):
        run(t)
        torch.cuda.synchronize()
        eager.append(dw.tokens.clone())
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        run(20)
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    outs = [torch.empty_like(dw.tokens) for _ in range(3)]
    with torch.cuda.graph(g, stream=s):
        for j, t in enumerate((20, 21, 22)):
            run(t)
            outs[j].copy_(dw.tokens)
    for _ in range(2):
        g.replay()
        torch.cuda.synchronize()
        for j in range(3):
            assert torch.equal(outs[j], eager[j])
    dw.check_no_device_error()
