"""ctypes binding of the fp64 CPU oracle (oracle/cfgms_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cfgms_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

FLAG_INACTIVE, FLAG_GREEDY, FLAG_CLOSE, FLAG_BOUNDARY, FLAG_FORCED = 1, 2, 4, 8, 16
TOL = 2e-2  # north_star's margin below which a tie is "close" (counted, not failed)


# CFGMS_ORACLE_SANITIZE=1 (tests/test_oracle_sanitizers.py sets it for a child process that preloads the ASan
# runtime): the same source built with AddressSanitizer + UndefinedBehaviorSanitizer into a library of its own.
_SANITIZE = os.environ.get("CFGMS_ORACLE_SANITIZE", "") == "1"
if _SANITIZE:
    _LIB = os.path.join(_HERE, "liboracle_san.so")


def build(force: bool = False) -> str:
    """gcc -O2, no fast-math, no FMA contraction: the fp64 sums keep the written order."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off"]
        if _SANITIZE:   # same arithmetic (no contraction, same order); -O1 and frame pointers for readable reports
            cmd = ["gcc", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                   "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off"]
        subprocess.run(cmd + ["-o", _LIB, _SRC, "-lm"], check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_uniform.restype = C.c_double
        L.oracle_uniform.argtypes = [C.c_uint32]
        L.oracle_gumbel_from_uniform.restype = C.c_double
        L.oracle_gumbel_from_uniform.argtypes = [C.c_double]
        L.oracle_gumbel.restype = C.c_double
        L.oracle_gumbel.argtypes = [C.c_uint64, C.c_uint32, C.c_int32, C.c_int32, C.c_int32]
        L.oracle_sample_cell.restype = C.c_int32
        L.oracle_sample_cell.argtypes = [C.c_void_p, C.c_int32, C.c_float, C.c_int32, C.c_uint64,
                                         C.c_uint32, C.c_int32, C.c_int32, C.c_double,
                                         C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_step.restype = C.c_int
        L.oracle_step.argtypes = ([C.c_void_p] * 3 + [C.c_int32] * 4 + [C.c_void_p] * 4 + [C.c_uint64]
                                  + [C.c_void_p] * 3 + [C.c_int32, C.c_double, C.c_void_p, C.c_int64]
                                  + [C.c_void_p] * 6 + [C.c_int32])
        L.oracle_step_ex.restype = C.c_int
        L.oracle_step_ex.argtypes = L.oracle_step.argtypes + [C.c_void_p, C.c_void_p]
        L.oracle_emit_frame.restype = C.c_int32
        L.oracle_emit_frame.argtypes = [C.c_void_p] + [C.c_int32] * 5 + [C.c_void_p]
        L.oracle_feedback.restype = None
        L.oracle_feedback.argtypes = [C.c_void_p, C.c_void_p] + [C.c_int32] * 4 + [C.c_void_p]
        L.oracle_advance_state.restype = C.c_int32
        L.oracle_advance_state.argtypes = [C.c_int32] * 6 + [C.c_void_p, C.c_void_p]
        L.oracle_phase_advance.restype = C.c_int32
        L.oracle_phase_advance.argtypes = [C.c_int32] * 9 + [C.c_void_p] * 3
        L.oracle_step_phase.restype = C.c_int
        L.oracle_step_phase.argtypes = ([C.c_void_p] * 3 + [C.c_int32] * 4 + [C.c_void_p] * 4 + [C.c_uint64]
                                        + [C.c_void_p] * 3 + [C.c_int32, C.c_double, C.c_void_p, C.c_int64]
                                        + [C.c_void_p] * 6 + [C.c_int32] + [C.c_void_p] * 3 + [C.c_int32, C.c_void_p, C.c_int32,
                                                                                                C.c_void_p])
        L.oracle_logits_row.restype = None
        L.oracle_logits_row.argtypes = [C.c_void_p] * 3 + [C.c_int32] * 5 + [C.c_void_p]
        L.oracle_cfg_merge.restype = None
        L.oracle_cfg_merge.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_int32, C.c_void_p]
        L.oracle_deinterleave.restype = C.c_int
        L.oracle_deinterleave.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.oracle_interleave.restype = C.c_int
        L.oracle_interleave.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.oracle_sample_sweep.restype = None
        L.oracle_sample_sweep.argtypes = [C.c_void_p, C.c_int32, C.c_float, C.c_int32, C.c_uint64,
                                          C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.oracle_check_pair_map.restype = C.c_int
        L.oracle_check_pair_map.argtypes = [C.c_void_p, C.c_int32]
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _arr(a, dtype) -> Optional[np.ndarray]:
    if a is None:
        return None
    if hasattr(a, "detach"):  # torch tensor (bf16 goes through its int16 bit view)
        import torch
        a = a.detach().cpu()
        if a.dtype == torch.bfloat16:
            a = a.contiguous().view(torch.int16)
        a = a.numpy()
    a = np.asarray(a)
    if dtype == np.uint16 and a.dtype == np.int16:
        a = a.view(np.uint16)
    if dtype == np.uint32 and a.dtype == np.int32:
        a = a.view(np.uint32)
    return np.ascontiguousarray(a, dtype=dtype)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def bf16_to_f64(bits) -> np.ndarray:
    b = _arr(bits, np.uint16)
    out = np.empty(b.shape, dtype=np.float64)
    lib().oracle_bf16_to_f64(_p(b), C.c_int64(b.size), _p(out))
    return out


def f32_to_bf16(x) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round to nearest even (reading C18)."""
    f = _arr(x, np.float32)
    out = np.empty(f.shape, dtype=np.uint16)
    lib().oracle_f32_to_bf16_rne(_p(f), C.c_int64(f.size), _p(out))
    return out


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def uniform(x: int) -> float:
    return float(lib().oracle_uniform(C.c_uint32(int(x))))


def gumbel(seed: int, req_id: int, tau: int, stream: int, v: int) -> float:
    return float(lib().oracle_gumbel(C.c_uint64(seed), C.c_uint32(req_id), tau, stream, v))


def logits_row(heads, embeds, hidden, row: int, stream: int) -> np.ndarray:
    h = _arr(heads, np.uint16)
    e = _arr(embeds, np.uint16)
    x = _arr(hidden, np.uint16)
    S, V, d = h.shape
    out = np.empty(V, dtype=np.float64)
    lib().oracle_logits_row(_p(h), _p(e), _p(x), S, d, V, row, stream, _p(out))
    return out


def cfg_merge(l_cond, l_uncond, w: float) -> np.ndarray:
    a = np.ascontiguousarray(l_cond, dtype=np.float64)
    b = np.ascontiguousarray(l_uncond, dtype=np.float64)
    out = np.empty_like(a)
    lib().oracle_cfg_merge(_p(a), _p(b), C.c_double(w), a.size, _p(out))
    return out


def sample_cell(M, temp: float, top_k: int, seed: int, req_id: int, tau: int, stream: int,
                tol: float = TOL):
    """-> (token, margin, flags, thr)"""
    m = np.ascontiguousarray(M, dtype=np.float64)
    margin = C.c_double()
    flags = C.c_int32()
    thr = C.c_double()
    tok = lib().oracle_sample_cell(_p(m), m.size, C.c_float(temp), top_k, C.c_uint64(seed),
                                   C.c_uint32(req_id), tau, stream, C.c_double(tol),
                                   C.byref(margin), C.byref(flags), C.byref(thr))
    return int(tok), float(margin.value), int(flags.value), float(thr.value)


def sample_sweep(M, temp: float, top_k: int, seed: int, n_req: int, n_tau: int, stream: int = 0) -> np.ndarray:
    """Token counts over n_req * n_tau independent draws of O6-O8 on fixed logits (test helper)."""
    m = np.ascontiguousarray(M, dtype=np.float64)
    counts = np.zeros(m.size, dtype=np.int64)
    lib().oracle_sample_sweep(_p(m), m.size, C.c_float(temp), top_k, C.c_uint64(seed), n_req, n_tau,
                              stream, _p(counts))
    return counts


class StepResult:
    __slots__ = ("cells", "tok", "margin", "flags", "merged", "tokens_out", "delayed")


def step(heads, embeds, hidden, pair_map, w, temp, top_k, seed: int, step_, req_id=None,
         n_frames=None, pad_token: Optional[int] = None, cells=None, want_merged: bool = False,
         tokens_out: Optional[np.ndarray] = None, delayed: Optional[np.ndarray] = None,
         tol: float = TOL, hidden_is_f32: bool = False, logit_bias=None, force_token=None) -> StepResult:
    """One decode step (O1-O10).  `hidden` is bf16 (torch) or, with hidden_is_f32, fp32 that is
    first rounded to bf16 (C18).  `cells` = None (all) or int array [n][2] of (row, stream)."""
    h = _arr(heads, np.uint16)
    e = _arr(embeds, np.uint16)
    x = f32_to_bf16(hidden) if hidden_is_f32 else _arr(hidden, np.uint16)
    S, V, d = h.shape
    R = x.shape[0]
    pm = _arr(pair_map, np.int32)
    ww = _arr(w, np.float32)
    tt = _arr(temp, np.float32)
    kk = _arr(top_k, np.int32)
    st = _arr(step_, np.int32)
    rid = _arr(req_id, np.uint32)
    nf = _arr(n_frames, np.int32)
    pad = V if pad_token is None else int(pad_token)
    if cells is None:
        rows = [r for r in range(R) if pm[r] < 0 or r % 2 == 0]
        cl = np.asarray([(r, i) for r in rows for i in range(S)], dtype=np.int32).reshape(-1, 2)
    else:
        cl = np.ascontiguousarray(cells, dtype=np.int32).reshape(-1, 2)
    n = cl.shape[0]
    res = StepResult()
    res.cells = cl
    res.tok = np.empty(n, dtype=np.int32)
    res.margin = np.empty(n, dtype=np.float64)
    res.flags = np.empty(n, dtype=np.int32)
    res.merged = np.empty((n, V), dtype=np.float64) if want_merged else None
    res.tokens_out = tokens_out
    res.delayed = delayed
    T_cap = 0
    if delayed is not None:
        assert delayed.dtype == np.int32 and delayed.flags.c_contiguous and delayed.shape[0] == R
        T_cap = delayed.shape[1]
    if tokens_out is not None:
        assert tokens_out.dtype == np.int32 and tokens_out.flags.c_contiguous
    lb = _arr(logit_bias, np.float64)     # widening W2: [S][V] additive bias (-inf masks a token)
    ft = _arr(force_token, np.int32)      # widening W2: [R][S], >= 0 forces the cell's token
    if lb is not None:
        assert lb.shape == (S, V)
    if ft is not None:
        assert ft.shape == (R, S)
    rc = lib().oracle_step_ex(_p(h), _p(e), _p(x), R, S, d, V, _p(pm), _p(ww), _p(tt), _p(kk),
                              C.c_uint64(seed), _p(st), _p(rid), _p(nf), pad, C.c_double(tol),
                              _p(cl), C.c_int64(n), _p(res.tok), _p(res.margin), _p(res.flags),
                              _p(res.merged), _p(tokens_out), _p(delayed), T_cap, _p(lb), _p(ft))
    if rc != 0:
        raise ValueError(f"oracle_step failed with code {rc}")
    return res


def check_pair_map(pair_map) -> int:
    pm = _arr(pair_map, np.int32)
    return int(lib().oracle_check_pair_map(_p(pm), pm.size))


def deinterleave(delayed: np.ndarray) -> np.ndarray:
    """[n][T][S] int32 -> [n][T-S+1][S]"""
    dl = np.ascontiguousarray(delayed, dtype=np.int32)
    n, T, S = dl.shape
    grid = np.empty((n, T - S + 1, S), dtype=np.int32)
    rc = lib().oracle_deinterleave(_p(dl), n, T, S, _p(grid))
    if rc != 0:
        raise ValueError(f"oracle_deinterleave failed with code {rc}")
    return grid


def interleave(grid: np.ndarray, pad: int) -> np.ndarray:
    """[n][F][S] int32 -> [n][F+S-1][S] with PAD in the S(S-1)/2 head and tail cells"""
    g = np.ascontiguousarray(grid, dtype=np.int32)
    n, F, S = g.shape
    dl = np.empty((n, F + S - 1, S), dtype=np.int32)
    rc = lib().oracle_interleave(_p(g), n, F, S, int(pad), _p(dl))
    if rc != 0:
        raise ValueError(f"oracle_interleave failed with code {rc}")
    return dl


def emit_frame(ring: np.ndarray, tau: int, n_frames: int, pad: int):
    """Widening W1.  ring: int32 [T_cap][S] of ONE request (ring[t % T_cap][i] = token of stream i
    at step t).  -> (frame index or -1, frame int32 [S])."""
    rg = np.ascontiguousarray(ring, dtype=np.int32)
    T_cap, S = rg.shape
    frame = np.empty(S, dtype=np.int32)
    f = lib().oracle_emit_frame(_p(rg), T_cap, S, int(tau), int(n_frames), int(pad), _p(frame))
    return int(f), frame


def feedback(tokens, emb) -> np.ndarray:
    """Widening W3.  tokens int32 [R][S], emb bf16 [S][V_e][d] -> float64 [R][d] (exact sums)."""
    tk = _arr(tokens, np.int32)
    eb = _arr(emb, np.uint16)
    R, S = tk.shape
    S2, V_e, d = eb.shape
    assert S == S2
    x = np.empty((R, d), dtype=np.float64)
    lib().oracle_feedback(_p(tk), _p(eb), R, S, V_e, d, _p(x))
    return x


F_UNSET = 2 ** 31 - 1   # "no frame count yet": every stream i <= tau stays active


def advance_state(tau: int, F: int, tok0: int, eos: int, S: int):
    """Widening W4 -> (tau_next, F_next, drained)."""
    tn, fn = C.c_int32(), C.c_int32()
    done = lib().oracle_advance_state(int(tau), int(F), int(tok0), int(eos), int(S), F_UNSET, C.byref(tn), C.byref(fn))
    return int(tn.value), int(fn.value), bool(done)


# ---- widening W6: per-request phase state machine (readings C28-C32) ----
PHASE_TEXT, PHASE_TRANSITION, PHASE_AUDIO, PHASE_DONE = 0, 1, 2, 3


def phase_advance(phase: int, pos: int, F: int, tok0: int, modality_audio: bool, n_bridge: int, eos: int, S: int):
    """One transition of the phase state machine -> (phase_next, pos_next, F_next, done)."""
    pn, qn, fn = C.c_int32(), C.c_int32(), C.c_int32()
    done = lib().oracle_phase_advance(int(phase), int(pos), int(F), int(tok0), int(bool(modality_audio)), int(n_bridge),
                                      int(eos), int(S), F_UNSET, C.byref(pn), C.byref(qn), C.byref(fn))
    return int(pn.value), int(qn.value), int(fn.value), bool(done)


class PhaseStepResult(StepResult):
    __slots__ = ("modality",)


def step_phase(heads, embeds, hidden, pair_map, w, temp, top_k, seed: int, gstep, phase, pos, V_text: int, bridge,
               req_id=None, n_frames=None, pad_token: Optional[int] = None, cells=None, want_merged: bool = False,
               tokens_out: Optional[np.ndarray] = None, delayed: Optional[np.ndarray] = None, tol: float = TOL,
               hidden_is_f32: bool = False, logit_bias=None) -> PhaseStepResult:
    """One decode step of a batch whose requests sit in different phases (oracle_step_phase).  `gstep` is the
    request's global step (noise key); `pos` the bridging position (TRANSITION) or audio-local step (AUDIO)."""
    h = _arr(heads, np.uint16)
    e = _arr(embeds, np.uint16)
    x = f32_to_bf16(hidden) if hidden_is_f32 else _arr(hidden, np.uint16)
    S, V, d = h.shape
    R = x.shape[0]
    pm = _arr(pair_map, np.int32)
    ww, tt, kk = _arr(w, np.float32), _arr(temp, np.float32), _arr(top_k, np.int32)
    st, ph, ps = _arr(gstep, np.int32), _arr(phase, np.int32), _arr(pos, np.int32)
    rid, nf = _arr(req_id, np.uint32), _arr(n_frames, np.int32)
    br = np.ascontiguousarray(bridge, dtype=np.int32).reshape(-1)
    pad = V if pad_token is None else int(pad_token)
    if cells is None:
        rows = [r for r in range(R) if pm[r] < 0 or r % 2 == 0]
        cl = np.asarray([(r, i) for r in rows for i in range(S)], dtype=np.int32).reshape(-1, 2)
    else:
        cl = np.ascontiguousarray(cells, dtype=np.int32).reshape(-1, 2)
    n = cl.shape[0]
    res = PhaseStepResult()
    res.cells = cl
    res.tok = np.empty(n, dtype=np.int32)
    res.margin = np.empty(n, dtype=np.float64)
    res.flags = np.empty(n, dtype=np.int32)
    res.modality = np.zeros(n, dtype=np.int32)
    res.merged = np.empty((n, V), dtype=np.float64) if want_merged else None
    res.tokens_out, res.delayed = tokens_out, delayed
    T_cap = 0
    if delayed is not None:
        assert delayed.dtype == np.int32 and delayed.flags.c_contiguous and delayed.shape[0] == R
        T_cap = delayed.shape[1]
    lb = _arr(logit_bias, np.float64)
    rc = lib().oracle_step_phase(_p(h), _p(e), _p(x), R, S, d, V, _p(pm), _p(ww), _p(tt), _p(kk), C.c_uint64(seed),
                                 _p(st), _p(rid), _p(nf), pad, C.c_double(tol), _p(cl), C.c_int64(n), _p(res.tok),
                                 _p(res.margin), _p(res.flags), _p(res.merged), _p(tokens_out), _p(delayed), T_cap, _p(lb),
                                 _p(ph), _p(ps), int(V_text), _p(br), int(br.size), _p(res.modality))
    if rc != 0:
        raise ValueError(f"oracle_step_phase failed with code {rc}")
    return res
