"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

This module is the ONLY code shared by the oracle-side tests and the CUDA path.  It holds
none of the method's arithmetic: it draws Gaussian / uniform tensors from named, seeded
torch CPU generators, rounds them to bf16 (RNE, input preparation) and lays the batch out
as the paper's Paired Request Co-Scheduling would (section 2.4: the
conditional row sits next to its unconditional companion in one continuous batch).

Readings applied:
  * N(0, x): x is a variance            (hidden std 1, heads std d**-0.5, embeds std sqrt(0.02))
  * config 3 heavy tail: round(0.01*V) columns per stream get an extra N(0, 9/d)^d vector added
    to the head row before bf16 rounding -> every raw logit at that column gains 3*N(0,1)
  * config 4: 192 two-row slots in seeded order: 128 (cond, uncond) pairs + 64 slots holding
    two unpaired rows; request q has start offset o_q in [0, S) and local step tau = t + o_q
  * hidden states of step t come from a pool of P independent batches: pool[t % P]

The paper's own workloads (LibriSpeech TTS / MMAU-mini / Eval2000 through Bagpiper, OpusLM,
OpusLM-Dialogue) are not available; these batches stand in for their
shapes (S = 8/16 streams, d = 2048/4096, 128-1024 concurrent rows).
"""
from __future__ import annotations

import zlib
from dataclasses import dataclass, field
from typing import Optional

import numpy as np
import torch

# (name, B pairs, unpaired rows, d, S, V, hidden dtype, w, temp, top_k, T)
CONFIGS = {
    1: dict(name="tiny", pairs=2, singles=0, d=256, S=4, V=256, hidden_f32=True,
            w=3.0, temp=1.0, top_k=16, T=24),
    2: dict(name="mid", pairs=64, singles=0, d=2048, S=8, V=1024, hidden_f32=False,
            w=3.0, temp=0.8, top_k=50, T=256),
    3: dict(name="7b_head", pairs=128, singles=0, d=4096, S=8, V=4096, hidden_f32=False,
            w=2.0, temp=0.9, top_k=100, T=512, heavy_tail=True),
    4: dict(name="mixed", pairs=128, singles=128, d=4096, S=8, V=2048, hidden_f32=False,
            w=None, temp=None, top_k=None, T=256, mixed=True),
    5: dict(name="large", pairs=512, singles=0, d=4096, S=16, V=2048, hidden_f32=False,
            w=3.0, temp=1.0, top_k=50, T=1024),
}


def _gen(base_seed: int, name: str) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed((int(base_seed) * 1000003 + zlib.crc32(name.encode())) % (2 ** 63))
    return g


@dataclass
class Workload:
    """One synthetic batch description. All tensors live on the CPU; callers upload."""
    cfg: int
    name: str
    R: int
    n_req: int
    d: int
    S: int
    V: int
    T: int
    seed: int
    heads: torch.Tensor            # bf16 [S][V][d]
    embeds: torch.Tensor           # bf16 [S][d]
    hidden_pool: torch.Tensor      # [P][R][d], fp32 for config 1 else bf16
    pair_map: torch.Tensor         # int32 [R]
    w: torch.Tensor                # fp32 [R]  (read at cond rows)
    temp: torch.Tensor             # fp32 [R]
    top_k: torch.Tensor            # int32 [R]
    req_id: torch.Tensor           # int32 [R] (bit pattern of uint32)
    n_frames: Optional[torch.Tensor]   # int32 [R] or None
    offset: torch.Tensor           # int32 [R] start offset o_q (0 except config 4)
    pad_token: int = field(default=0)

    @property
    def hidden_f32(self) -> bool:
        return self.hidden_pool.dtype == torch.float32

    def hidden(self, t: int) -> torch.Tensor:
        return self.hidden_pool[t % self.hidden_pool.shape[0]]

    def step(self, t: int) -> torch.Tensor:
        """Request-local decode step tau of every row at engine iteration t."""
        return (self.offset + int(t)).to(torch.int32)

    def head_rows(self) -> np.ndarray:
        """Batch rows that own a request (cond rows of pairs and unpaired rows)."""
        pm = self.pair_map.numpy()
        rows = [r for r in range(self.R) if pm[r] < 0 or (r % 2 == 0 and pm[r] == r + 1)]
        return np.asarray(rows, dtype=np.int32)


def _layout(pairs: int, singles: int, base_seed: int, shuffle: bool):
    """Two-row slots: a slot is one (cond, uncond) pair or two unpaired rows."""
    assert singles % 2 == 0
    kinds = [1] * pairs + [0] * (singles // 2)
    if shuffle:
        perm = torch.randperm(len(kinds), generator=_gen(base_seed, "slot_order")).tolist()
        kinds = [kinds[p] for p in perm]
    R = 2 * len(kinds)
    pair_map = np.full(R, -1, dtype=np.int32)
    for s, kind in enumerate(kinds):
        if kind:
            pair_map[2 * s] = 2 * s + 1
            pair_map[2 * s + 1] = 2 * s
    return R, pair_map


def make_config(cfg: int, base_seed: int = 0, pool: int = 8, cfg_off: bool = False,
                overrides: Optional[dict] = None) -> Workload:
    """Build config `cfg` (1..5).  cfg_off=True gives the CFG-off twin of BASELINE.json
    configs[1]: the same cond rows only, every row its own request (pair_map = -1)."""
    c = dict(CONFIGS[cfg])
    if overrides:
        c.update(overrides)
    d, S, V, T = c["d"], c["S"], c["V"], c["T"]
    pairs, singles = c["pairs"], c["singles"]
    mixed = bool(c.get("mixed"))

    R, pair_map = _layout(pairs, singles, base_seed, shuffle=mixed)
    n_req = pairs + singles

    heads = torch.randn(S, V, d, generator=_gen(base_seed, "heads")) * (d ** -0.5)
    if c.get("heavy_tail"):
        ncol = int(round(0.01 * V))
        for i in range(S):
            cols = torch.randperm(V, generator=_gen(base_seed, f"tail_cols_{i}"))[:ncol]
            extra = torch.randn(ncol, d, generator=_gen(base_seed, f"tail_vals_{i}")) * (3.0 * d ** -0.5)
            heads[i, cols] += extra
    heads = heads.to(torch.bfloat16)
    embeds = (torch.randn(S, d, generator=_gen(base_seed, "embeds")) * (0.02 ** 0.5)).to(torch.bfloat16)
    hidden_pool = torch.randn(pool, R, d, generator=_gen(base_seed, "hidden"))
    if not c["hidden_f32"]:
        hidden_pool = hidden_pool.to(torch.bfloat16)

    w = torch.ones(R, dtype=torch.float32)
    temp = torch.ones(R, dtype=torch.float32)
    top_k = torch.zeros(R, dtype=torch.int32)
    offset = torch.zeros(R, dtype=torch.int32)
    req_id = torch.zeros(R, dtype=torch.int32)
    heads_rows = [r for r in range(R) if pair_map[r] < 0 or r % 2 == 0]
    if mixed:
        gw = _gen(base_seed, "w")
        gt = _gen(base_seed, "temp")
        gk = _gen(base_seed, "top_k")
        go = _gen(base_seed, "offset")
        choices = torch.tensor([1, 20, 50], dtype=torch.int32)
        for q, r in enumerate(heads_rows):
            if pair_map[r] >= 0:
                w[r] = 1.0 + 4.0 * torch.rand((), generator=gw)
            temp[r] = 0.6 + 0.6 * torch.rand((), generator=gt)
            top_k[r] = choices[torch.randint(0, 3, (), generator=gk)]
            offset[r] = torch.randint(0, S, (), generator=go)
            req_id[r] = q
        n_frames = None
    else:
        for q, r in enumerate(heads_rows):
            w[r] = c["w"]
            temp[r] = c["temp"]
            top_k[r] = c["top_k"]
            req_id[r] = q
        n_frames = torch.full((R,), T - S + 1, dtype=torch.int32)
    # companions carry a copy of their cond row's parameters (they are ignored, reading C14)
    for r in range(R):
        if pair_map[r] >= 0 and r % 2 == 1:
            for a in (w, temp, top_k, offset, req_id):
                a[r] = a[r - 1]

    wl = Workload(cfg=cfg, name=c["name"], R=R, n_req=n_req, d=d, S=S, V=V, T=T, seed=base_seed,
                  heads=heads, embeds=embeds, hidden_pool=hidden_pool,
                  pair_map=torch.from_numpy(pair_map), w=w, temp=temp, top_k=top_k,
                  req_id=req_id, n_frames=n_frames, offset=offset, pad_token=V)
    if cfg_off:
        wl = cfg_off_twin(wl)
    return wl


def cfg_off_twin(wl: Workload) -> Workload:
    """Keep only request-owning rows; every row becomes an unpaired request (CFG off)."""
    rows = torch.from_numpy(wl.head_rows().astype(np.int64))
    sel = lambda a: None if a is None else a[rows].clone()
    R = int(rows.numel())
    return Workload(cfg=wl.cfg, name=wl.name + "_cfg_off", R=R, n_req=R, d=wl.d, S=wl.S, V=wl.V,
                    T=wl.T, seed=wl.seed, heads=wl.heads, embeds=wl.embeds,
                    hidden_pool=wl.hidden_pool[:, rows].clone(),
                    pair_map=torch.full((R,), -1, dtype=torch.int32),
                    w=torch.ones(R, dtype=torch.float32), temp=sel(wl.temp), top_k=sel(wl.top_k),
                    req_id=sel(wl.req_id), n_frames=sel(wl.n_frames), offset=sel(wl.offset),
                    pad_token=wl.pad_token)


def parity_steps(cfg: int, T: int, S: int) -> list:
    """Engine iterations the parity tests check (head, drain tail, two seeded mid points)."""
    if cfg == 1:
        return list(range(T))
    g = _gen(0, f"parity_steps_{cfg}")
    mid = [int(torch.randint(S, T - S, (), generator=g)) for _ in range(2)]
    if cfg == 2:
        base = list(range(0, S + 1)) + list(range(T - S - 1, T))
    elif cfg == 3:
        base = [0, S - 1, S, T - S, T - 1]
    elif cfg == 4:
        base = [0, 1, S - 1, S, T - 1]
    else:
        base = [0, S - 1, T - 1]
    return sorted(set(base + mid[: (2 if cfg == 2 else 1)]))
