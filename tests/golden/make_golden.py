"""Writes tests/golden/config1_oracle.txt: the oracle's tokens, PAD pattern and de-interleaved
code grid for BASELINE.json configs[0] (tiny: 2 CFG pairs, S = 4, V = 256, 24 steps, seed 0).

The paper prints no worked numeric example ("whole step: parity unpinned"), so
this file is NOT a paper value: it is a regression fixture written by this script, which calls only
oracle/ and the seeded input generators of workloads.py.  It freezes the oracle's behaviour so that a
later change to its arithmetic (or to the input recipe) cannot slip by unnoticed, and gives the GPU
tests a stored expectation that never came from the CUDA path.

    python tests/golden/make_golden.py          # rewrites the fixture
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")


def compute():
    wl = workloads.make_config(1)
    delayed = np.full((wl.R, wl.T, wl.S), -1, dtype=np.int32)
    close = []
    for t in range(wl.T):
        res = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                          wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, delayed=delayed,
                          hidden_is_f32=wl.hidden_f32)
        for j, (c, i) in enumerate(res.cells):
            if res.flags[j] & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
                close.append((t, int(c), int(i)))
    heads = wl.head_rows()
    grid = oracle.deinterleave(delayed[heads])
    return wl, heads, delayed, grid, close


def render():
    wl, heads, delayed, grid, close = compute()
    lines = ["# oracle fixture, BASELINE.json configs[0]; written by tests/golden/make_golden.py (calls only oracle/)",
             f"# R={wl.R} S={wl.S} V={wl.V} d={wl.d} T={wl.T} pad={wl.pad_token} seed={wl.seed}",
             "# delayed <request row> <step> : S tokens (PAD = %d)" % wl.pad_token]
    for c in heads:
        for t in range(wl.T):
            lines.append(f"delayed {int(c)} {t} : " + " ".join(str(int(x)) for x in delayed[c, t]))
    lines.append("# grid <request index> <frame> : S codes")
    for q in range(grid.shape[0]):
        for f in range(grid.shape[1]):
            lines.append(f"grid {q} {f} : " + " ".join(str(int(x)) for x in grid[q, f]))
    lines.append("# close <step> <row> <stream> : cells the oracle flags as close ties (margin <= 2e-2 or top-k edge)")
    for t, c, i in close:
        lines.append(f"close {t} {c} {i}")
    return "\n".join(lines) + "\n"


if __name__ == "__main__":
    with open(OUT, "w") as f:
        f.write(render())
    print("wrote", OUT)
