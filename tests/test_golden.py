"""tests/golden/config1_oracle.txt (written by tests/golden/make_golden.py from oracle/ alone):
the oracle must still reproduce it (CPU), and the CUDA path must reproduce it outside the cells the
oracle itself flags as close ties (GPU)."""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
FIXTURE = os.path.join(HERE, "golden", "config1_oracle.txt")


def _load():
    delayed, grid, close = {}, {}, set()
    for line in open(FIXTURE):
        if line.startswith("#") or not line.strip():
            continue
        head, _, tail = line.partition(":")
        parts = head.split()
        if parts[0] == "delayed":
            delayed[(int(parts[1]), int(parts[2]))] = [int(x) for x in tail.split()]
        elif parts[0] == "grid":
            grid[(int(parts[1]), int(parts[2]))] = [int(x) for x in tail.split()]
        elif parts[0] == "close":
            close.add((int(parts[1]), int(parts[2]), int(parts[3])))
    return delayed, grid, close


def test_oracle_still_writes_the_fixture():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    assert mod.render() == open(FIXTURE).read()


def test_fixture_has_the_delay_pattern_of_the_paper():
    # PAPER.md:56,76 + BASELINE north_star: stream i lags i steps, PAD in the first S-1 and last S-1 steps,
    # interleave . de-interleave = identity
    delayed, grid, _ = _load()
    S, T, pad = 4, 24, 256
    F = T - S + 1
    for c in (0, 2):
        q = c // 2
        for t in range(T):
            for i in range(S):
                f = t - i
                if 0 <= f < F:
                    assert delayed[(c, t)][i] == grid[(q, f)][i] != pad
                else:
                    assert delayed[(c, t)][i] == pad


@pytest.mark.gpu
def test_cuda_path_reproduces_the_fixture():
    import torch

    import workloads
    from parity_util import DeviceWorkload
    delayed, grid, close = _load()
    wl = workloads.make_config(1)
    dw = DeviceWorkload(wl, torch.device("cuda:0"))
    for t in range(wl.T):
        dw.step(t)
    dw.check_no_device_error()
    got = dw.delayed.cpu().numpy()
    for (c, t), want in delayed.items():
        for i, tok in enumerate(want):
            if (t, c, i) not in close:
                assert got[c, t, i] == tok, (c, t, i)
    heads = torch.from_numpy(wl.head_rows().astype(np.int64)).to(dw.dev)
    g = dw.ctx.deinterleave(dw.delayed[heads].contiguous()).cpu().numpy()
    for (q, f), want in grid.items():
        for i, code in enumerate(want):
            if (f + i, int(wl.head_rows()[q]), i) not in close:
                assert g[q, f, i] == code, (q, f, i)
