"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md test strategy: "oracle built with
-fsanitize=address,undefined in a test target").  Every parity claim rests on oracle/cfgms_oracle.c, so its own memory
safety is checked once, on the CPU: a child process preloads the ASan runtime, builds the same source with both
sanitizers (oracle/__init__.py, CFGMS_ORACLE_SANITIZE=1) and drives every entry point the parity tests use — a full
config-1 step, a phase-machine step with an empty region, ragged delay round trips, frame emission, feedback with
out-of-range ids — and prints a digest; the digest must equal the regular build's (same arithmetic, same order), and
any sanitizer report aborts the child."""
import hashlib
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r'''
import hashlib, sys
import numpy as np
sys.path.insert(0, %r)
import oracle, workloads
h = hashlib.sha256()
def eat(*arrs):
    for a in arrs:
        h.update(np.ascontiguousarray(a).tobytes())
wl = workloads.make_config(1)
for t in (0, wl.S - 1, wl.S + 3):
    r = oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed, wl.step(t),
                    wl.req_id, wl.n_frames, wl.pad_token, want_merged=True, hidden_is_f32=wl.hidden_f32)
    eat(r.cells, r.tok, r.flags, r.margin, r.merged)
# odd shapes: V not a multiple of anything, S = 1, unpaired rows only; top_k at and beyond V
for ov in (dict(pairs=1, singles=2, d=24, S=3, V=37, T=8), dict(pairs=0, singles=2, d=8, S=1, V=5, T=4)):
    w2 = workloads.make_config(2, overrides=dict(mixed=True, hidden_f32=False, heavy_tail=False, **ov))
    r = oracle.step(w2.heads, w2.embeds, w2.hidden(1), w2.pair_map, w2.w, w2.temp, w2.top_k, w2.seed, w2.step(1),
                    w2.req_id, w2.n_frames, w2.pad_token)
    eat(r.tok, r.flags)
    ph = np.zeros(w2.R, dtype=np.int32); pos = np.zeros(w2.R, dtype=np.int32)
    for V_text in (0, 2):      # empty and non-empty text region
        r = oracle.step_phase(w2.heads, w2.embeds, w2.hidden(0), w2.pair_map, w2.w, w2.temp, w2.top_k, w2.seed,
                              np.arange(w2.R, dtype=np.int32), ph, pos, V_text, [1], req_id=w2.req_id, pad_token=w2.pad_token)
        eat(r.tok, r.flags, r.modality)
# delay pattern: interleave -> de-interleave round trip on ragged shapes, frame emission over a ring
rng = np.random.default_rng(3)
for (n, F, S) in ((1, 1, 1), (2, 5, 4), (3, 17, 9)):
    grid = rng.integers(0, 100, size=(n, F, S)).astype(np.int32)
    dl = oracle.interleave(grid, 1000)
    assert np.array_equal(oracle.deinterleave(dl), grid)
    eat(dl)
    for tau in range(F + S - 1):
        f, fr = oracle.emit_frame(dl[0], tau, F, 1000)
        eat(np.int32(f), fr)
tok = np.array([[0, 3, -1], [7, 2, 1]], dtype=np.int32)      # ids outside [0, V_e) contribute nothing
import torch
emb = torch.randn(3, 4, 16, generator=torch.Generator().manual_seed(1)).to(torch.bfloat16)
eat(oracle.feedback(tok, emb))
print("DIGEST", h.hexdigest())
''' % ROOT


def _run(env_extra):
    env = dict(os.environ, OMP_NUM_THREADS="4", **env_extra)
    return subprocess.run([sys.executable, "-c", DRIVER], env=env, capture_output=True, text=True, timeout=600)


def test_oracle_is_clean_under_asan_and_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("no ASan runtime in this toolchain")
    plain = _run({})
    assert plain.returncode == 0, plain.stderr[-2000:]
    san = _run({"CFGMS_ORACLE_SANITIZE": "1", "LD_PRELOAD": os.path.realpath(asan),
                "ASAN_OPTIONS": "detect_leaks=0:abort_on_error=1:halt_on_error=1", "UBSAN_OPTIONS": "halt_on_error=1:print_stacktrace=1"})
    assert san.returncode == 0, (san.stdout[-500:], san.stderr[-3000:])
    assert "ERROR: AddressSanitizer" not in san.stderr and "runtime error" not in san.stderr, san.stderr[-3000:]
    d0 = [l for l in plain.stdout.splitlines() if l.startswith("DIGEST")]
    d1 = [l for l in san.stdout.splitlines() if l.startswith("DIGEST")]
    assert d0 and d0 == d1
