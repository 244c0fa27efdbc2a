"""Shared helpers of the GPU parity tests: run the CUDA path through the C ABI on a seeded
workload and compare it, cell by cell, with the fp64 oracle.

Acceptance (BASELINE.json north_star, written here as the test's tolerance):
  * merged pre-temperature logits: max |gpu - oracle| <= 2e-2 (fp32 accumulate of bf16)
  * sampled token identical wherever the oracle's best-minus-second perturbed score > 2e-2
    and the outcome does not hinge on the top-k edge within 2e-2; closer ties are counted and
    reported, not failed
  * PAD cells, the companion row's copy, the delayed buffer and the de-interleaved grid:
    bit-exact
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
import workloads

LOGIT_TOL = 2e-2


class DeviceWorkload:
    def __init__(self, wl: workloads.Workload, dev, T_cap=None, row_tile: int = 0, no_candidates: bool = False,
                 no_overlap: bool = False, force_overlap: bool = False, **ctx_kwargs):
        import paper_2607_02119_b200 as pkg
        self.wl = wl
        self.dev = dev
        cu = lambda t: None if t is None else t.to(dev)
        self.heads = cu(wl.heads)
        self.embeds = cu(wl.embeds)
        self.ctx = pkg.Context(self.heads, self.embeds, max_rows=max(wl.R, 2), row_tile=row_tile,
                               no_candidates=no_candidates, no_overlap=no_overlap, force_overlap=force_overlap,
                               **ctx_kwargs)
        self.pool = cu(wl.hidden_pool)
        self.pair_map, self.w, self.temp, self.top_k = cu(wl.pair_map), cu(wl.w), cu(wl.temp), cu(wl.top_k)
        self.req_id, self.n_frames = cu(wl.req_id), cu(wl.n_frames)
        self.T_cap = wl.T if T_cap is None else T_cap
        self.delayed = torch.full((wl.R, self.T_cap, wl.S), -1, dtype=torch.int32, device=dev)
        self.tokens = torch.full((wl.R, wl.S), -1, dtype=torch.int32, device=dev)

    def hidden(self, t):
        return self.pool[t % self.pool.shape[0]]

    def step(self, t, logits_out=None, tokens=None):
        self.ctx.step(self.hidden(t), self.pair_map, self.w, self.temp, self.top_k, self.wl.seed,
                      self.wl.step(t).to(self.dev), self.tokens if tokens is None else tokens,
                      req_id=self.req_id, n_frames=self.n_frames, delayed=self.delayed, logits_out=logits_out)

    def check_no_device_error(self):
        torch.cuda.synchronize()
        rc, row = self.ctx.last_device_error()
        assert rc == 0, f"device error {rc} at row {row}"


def oracle_step(wl, t, cells=None, want_merged=True):
    return oracle.step(wl.heads, wl.embeds, wl.hidden(t), wl.pair_map, wl.w, wl.temp, wl.top_k, wl.seed,
                       wl.step(t), wl.req_id, wl.n_frames, wl.pad_token, cells=cells, want_merged=want_merged,
                       hidden_is_f32=wl.hidden_f32)


def sample_cells(wl, n_cells, seed):
    """Seeded subset of (request-owning row, stream) cells the oracle computes one by one."""
    rows = wl.head_rows()
    allc = np.asarray([(r, i) for r in rows for i in range(wl.S)], dtype=np.int32)
    if n_cells is None or n_cells >= len(allc):
        return allc
    rng = np.random.default_rng(seed)
    idx = np.sort(rng.choice(len(allc), size=n_cells, replace=False))
    return allc[idx]


CLOSE_FRAC_MAX = 0.03   # SURVEY 8(c) acceptance 2 expects 0.5-1.2 % close ties at the BASELINE shapes


def valid_alternative(wl, t, c, i, tok_gpu, logit_bias=None, tol=oracle.TOL):
    """For a cell the oracle flags close / boundary the GPU may pick another token — but only a
    token that a perturbation of z by < tol could have made win: it must lie inside the top-k
    set up to tol, `z[tok] >= thr - tol`, and its perturbed score must reach the oracle's best
    up to twice tol (both competitors may move), `z[tok] + g(tok) >= s_best - 2 tol`.  Greedy
    cells: `M[tok] >= max M - 2 tol`.  Recomputed from the oracle's own pieces for this one cell."""
    if not (0 <= tok_gpu < wl.V):
        return False
    hid = oracle.f32_to_bf16(wl.hidden(t)) if wl.hidden_f32 else wl.hidden(t)
    u = int(wl.pair_map[c])
    M = oracle.logits_row(wl.heads, wl.embeds, hid, int(c), int(i))
    if u >= 0:
        M = oracle.cfg_merge(M, oracle.logits_row(wl.heads, wl.embeds, hid, u, int(i)), float(wl.w[c]))
    if logit_bias is not None:
        M = M + np.asarray(logit_bias, dtype=np.float64)[i]
    temp, tk = float(wl.temp[c]), int(wl.top_k[c])
    tau = int(wl.step(t)[c])
    rid = int(wl.req_id[c]) & 0xFFFFFFFF
    tok, _, flags, thr = oracle.sample_cell(M, temp, tk, wl.seed, rid, tau, int(i), tol)
    if flags & oracle.FLAG_GREEDY:
        return bool(M[tok_gpu] >= M[tok] - 2 * tol)
    z = M / float(np.float32(temp))
    g = lambda v: oracle.gumbel(wl.seed, rid, tau, int(i), int(v))
    s_best = z[tok] + g(tok)
    return bool(z[tok_gpu] >= thr - tol and z[tok_gpu] + g(tok_gpu) >= s_best - 2 * tol)


class ParityStats:
    def __init__(self):
        self.n = self.n_pad = self.n_close = self.n_close_mismatch = self.n_tight_mismatch = 0
        self.max_logit_err = 0.0
        self.sq_err = 0.0
        self.n_logits = 0
        self.first_mismatch = None

    def assert_close_fraction(self, frac=CLOSE_FRAC_MAX, slack=2):
        """Close ties are counted and reported, not failed — but they must stay the rare event the
        margin statistics predict, and a differing close cell was already checked to hold a valid
        alternative (compare_step)."""
        n_sampled = self.n - self.n_pad
        assert self.n_close_mismatch <= self.n_close
        assert self.n_close <= frac * n_sampled + slack, f"{self.n_close} close ties among {n_sampled} sampled cells"

    def summary(self):
        rmse = (self.sq_err / max(self.n_logits, 1)) ** 0.5
        return (f"cells={self.n} pad={self.n_pad} close={self.n_close} close_mismatch={self.n_close_mismatch} "
                f"max_logit_err={self.max_logit_err:.3e} logit_rmse={rmse:.3e} first_mismatch={self.first_mismatch}")


def compare_step(dw: DeviceWorkload, t: int, cells, stats: ParityStats, check_logits=True):
    """Run step t on the GPU and compare the listed cells with the oracle."""
    wl = dw.wl
    logits = None
    if check_logits:
        logits = torch.zeros((wl.R, wl.S, wl.V), dtype=torch.float32, device=dw.dev)
    dw.tokens.fill_(-1)
    dw.step(t, logits_out=logits)
    dw.check_no_device_error()
    got = dw.tokens.cpu().numpy()
    ref = oracle_step(wl, t, cells=cells, want_merged=check_logits)
    pm = wl.pair_map.numpy()
    if check_logits:
        rows = torch.from_numpy(ref.cells[:, 0].astype(np.int64)).to(dw.dev)
        strs = torch.from_numpy(ref.cells[:, 1].astype(np.int64)).to(dw.dev)
        got_logits = logits[rows, strs].cpu().numpy().astype(np.float64)
    tau = wl.step(t).numpy()
    for j, (c, i) in enumerate(ref.cells):
        stats.n += 1
        fl = int(ref.flags[j])
        if pm[c] >= 0:
            assert got[pm[c], i] == got[c, i], f"companion row differs at step {t} row {c} stream {i}"
        dslot = int(tau[c]) % dw.T_cap
        if fl & oracle.FLAG_INACTIVE:
            stats.n_pad += 1
            assert got[c, i] == wl.pad_token, f"PAD expected at step {t} row {c} stream {i}, got {got[c, i]}"
            continue
        if check_logits:
            err = np.abs(got_logits[j] - ref.merged[j])
            stats.max_logit_err = max(stats.max_logit_err, float(err.max()))
            stats.sq_err += float((err ** 2).sum())
            stats.n_logits += err.size
            assert err.max() <= LOGIT_TOL, f"merged logits off by {err.max()} at step {t} row {c} stream {i}"
        assert 0 <= got[c, i] < wl.V
        if fl & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
            stats.n_close += 1
            if got[c, i] != ref.tok[j]:
                stats.n_close_mismatch += 1
                if stats.first_mismatch is None:
                    stats.first_mismatch = (t, int(c), int(i))
                assert valid_alternative(wl, t, c, i, int(got[c, i])), (
                    f"close cell at step {t} row {c} stream {i}: gpu token {got[c, i]} is not a valid alternative "
                    f"to the oracle's {ref.tok[j]} (margin {ref.margin[j]})")
        else:
            assert got[c, i] == ref.tok[j], (f"token mismatch at step {t} row {c} stream {i}: gpu {got[c, i]} "
                                             f"oracle {ref.tok[j]} margin {ref.margin[j]}")
    # the delayed buffer received exactly tokens_out at [row][tau mod T_cap]
    dl = dw.delayed.cpu().numpy()
    for c in wl.head_rows():
        assert np.array_equal(dl[c, int(tau[c]) % dw.T_cap], got[c])
    return got


def check_tokens_against_oracle(wl, t: int, got: np.ndarray) -> int:
    """A full [R][S] token matrix of step t (e.g. gathered from stream shards) against oracle.step: PAD and
    every cell outside the oracle's close / boundary flags bit-equal, a differing close cell a valid
    alternative, companion rows equal to their cond rows.  Returns the number of close cells."""
    ref = oracle_step(wl, t, want_merged=False)
    pm = wl.pair_map.numpy()
    n_close = 0
    for j, (c, i) in enumerate(ref.cells):
        fl = int(ref.flags[j])
        if pm[c] >= 0:
            assert got[pm[c], i] == got[c, i], (t, c, i)
        if fl & oracle.FLAG_INACTIVE:
            assert got[c, i] == wl.pad_token, (t, c, i, got[c, i])
        elif fl & (oracle.FLAG_CLOSE | oracle.FLAG_BOUNDARY):
            n_close += 1
            assert got[c, i] == ref.tok[j] or valid_alternative(wl, t, c, i, int(got[c, i])), (t, c, i, got[c, i], ref.tok[j])
        else:
            assert got[c, i] == ref.tok[j], (t, c, i, got[c, i], ref.tok[j], ref.margin[j])
    return n_close
