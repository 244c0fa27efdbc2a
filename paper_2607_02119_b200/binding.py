"""Thin ctypes binding of libcfgms.so (include/cfgms.h).  Argument marshalling only: every
step of the decode-head path runs in the library's sm_100a kernels.  torch is used for device
buffers and streams.  There is no fallback: a missing library raises at first use."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcfgms.so")

CFGMS_BF16, CFGMS_F32 = 0, 1
CFGMS_CFG_PAD_TOKEN = 1
CFGMS_CFG_NO_CANDIDATES = 2
CFGMS_CFG_SINGLE_CTA = 4
CFGMS_CFG_CTA_PAIR = 8
CFGMS_CFG_NO_OVERLAP = 16
CFGMS_CFG_OVERLAP = 32
CFGMS_CFG_NO_PDL_FINALIZE = 64
CFGMS_CFG_NO_SPLIT_K = 128
CFGMS_FRAMES_UNSET = 2 ** 31 - 1

STATUS = {0: "CFGMS_OK", 1: "CFGMS_ERR_ARG", 2: "CFGMS_ERR_SHAPE", 3: "CFGMS_ERR_LAYOUT", 4: "CFGMS_ERR_CUDA",
          5: "CFGMS_ERR_ARCH", 6: "CFGMS_ERR_NOMEM", 7: "CFGMS_ERR_TIMEOUT", 8: "CFGMS_ERR_LIMIT"}
CFGMS_ERR_LIMIT = 8
CFGMS_STATIC_SCRATCH_BYTES = 8 << 20

EXPORTS = ["cfgms_create", "cfgms_destroy", "cfgms_step", "cfgms_step_host", "cfgms_deinterleave",
           "cfgms_deinterleave_host", "cfgms_last_device_error", "cfgms_get_info", "cfgms_strerror",
           "cfgms_version", "cfgms_profile_enable", "cfgms_profile_read", "cfgms_overlap_stats",
           "cfgms_set_logit_bias", "cfgms_feedback", "cfgms_set_phase_table", "cfgms_exchange_create",
           "cfgms_exchange_connect", "cfgms_exchange_connect_ipc", "cfgms_exchange_wait", "cfgms_exchange_tokens",
           "cfgms_set_stream_vocab_sizes", "cfgms_deinterleave_host_static"]


class CfgmsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {STATUS.get(status, status)} ({_lib().cfgms_strerror(status).decode()})")


class cfgms_config(C.Structure):
    _fields_ = [("max_rows", C.c_int32), ("pad_token", C.c_int32), ("flags", C.c_uint32),
                ("row_tile", C.c_int32), ("max_stages", C.c_int32), ("stream_base", C.c_int32),
                ("stream_stride", C.c_int32), ("global_streams", C.c_int32)]


class cfgms_step_args(C.Structure):
    _fields_ = [("hidden", C.c_void_p), ("hidden_dtype", C.c_int32), ("R", C.c_int32),
                ("pair_map", C.c_void_p), ("w", C.c_void_p), ("temp", C.c_void_p), ("top_k", C.c_void_p),
                ("seed", C.c_uint64), ("step", C.c_void_p), ("req_id", C.c_void_p), ("n_frames", C.c_void_p),
                ("tokens_out", C.c_void_p), ("delayed", C.c_void_p), ("T_cap", C.c_int32),
                ("logits_out", C.c_void_p), ("force_token", C.c_void_p), ("frame_out", C.c_void_p),
                ("frame_index_out", C.c_void_p), ("eos_token", C.c_int32), ("step_next_out", C.c_void_p),
                ("n_frames_next_out", C.c_void_p), ("done_out", C.c_void_p), ("phase", C.c_void_p),
                ("phase_pos", C.c_void_p), ("phase_next_out", C.c_void_p), ("phase_pos_next_out", C.c_void_p),
                ("modality_out", C.c_void_p)]


class cfgms_info(C.Structure):
    _fields_ = [("S", C.c_int32), ("d", C.c_int32), ("V", C.c_int32), ("max_rows", C.c_int32),
                ("pad_token", C.c_int32), ("num_sms", C.c_int32), ("row_tile", C.c_int32),
                ("row_blocks", C.c_int32), ("vocab_tiles", C.c_int32), ("gemm_grid", C.c_int32),
                ("pipeline_stages", C.c_int32), ("launches_last_step", C.c_int32),
                ("launches_total", C.c_int64), ("h2d_bytes_last_step", C.c_int64),
                ("d2h_bytes_last_step", C.c_int64), ("cta_pair", C.c_int32), ("overlap", C.c_int32),
                ("split_k", C.c_int32), ("reserved0", C.c_int32)]


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with "
                               "`python -m paper_2607_02119_b200.build` (there is no fallback path)")
        L = C.CDLL(LIB_PATH)
        L.cfgms_create.restype = C.c_int
        L.cfgms_create.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
                                   C.POINTER(cfgms_config)]
        L.cfgms_destroy.restype = None
        L.cfgms_destroy.argtypes = [C.c_void_p]
        for name in ("cfgms_step", "cfgms_step_host"):
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = [C.c_void_p, C.POINTER(cfgms_step_args), C.c_void_p]
        for name in ("cfgms_deinterleave", "cfgms_deinterleave_host"):
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.cfgms_deinterleave_host_static.restype = C.c_int
        L.cfgms_deinterleave_host_static.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.cfgms_last_device_error.restype = C.c_int
        L.cfgms_last_device_error.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.cfgms_get_info.restype = C.c_int
        L.cfgms_get_info.argtypes = [C.c_void_p, C.POINTER(cfgms_info)]
        L.cfgms_profile_enable.restype = C.c_int
        L.cfgms_profile_enable.argtypes = [C.c_void_p, C.c_int]
        L.cfgms_profile_read.restype = C.c_int
        L.cfgms_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.cfgms_set_logit_bias.restype = C.c_int
        L.cfgms_set_logit_bias.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.cfgms_exchange_create.restype = C.c_int
        L.cfgms_exchange_create.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.POINTER(C.c_void_p)]
        L.cfgms_exchange_connect.restype = C.c_int
        L.cfgms_exchange_connect.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.cfgms_exchange_connect_ipc.restype = C.c_int
        L.cfgms_exchange_connect_ipc.argtypes = [C.c_void_p, C.c_void_p]
        L.cfgms_exchange_wait.restype = C.c_int
        L.cfgms_exchange_wait.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.cfgms_exchange_tokens.restype = C.c_int
        L.cfgms_exchange_tokens.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.cfgms_set_stream_vocab_sizes.restype = C.c_int
        L.cfgms_set_stream_vocab_sizes.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.c_void_p, C.c_void_p]
        L.cfgms_set_phase_table.restype = C.c_int
        L.cfgms_set_phase_table.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_int32]
        L.cfgms_feedback.restype = C.c_int
        L.cfgms_feedback.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.cfgms_overlap_stats.restype = C.c_int
        L.cfgms_overlap_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.cfgms_strerror.restype = C.c_char_p
        L.cfgms_strerror.argtypes = [C.c_int]
        L.cfgms_version.restype = C.c_char_p
        _LIB = L
    return _LIB


def library():
    """The loaded ctypes library (raises if libcfgms.so has not been built)."""
    return _lib()


def use_library(path: str) -> None:
    """Load another build of the library instead of libcfgms.so — the probe build of `bench.py --probes`
    (build.build_lib(probes=True)).  Must be called before the first library call of the process."""
    global LIB_PATH
    if _LIB is not None:
        raise RuntimeError("the library is already loaded")
    LIB_PATH = path


def version() -> str:
    return _lib().cfgms_version().decode()


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    return (stream if stream is not None else torch.cuda.current_stream()).cuda_stream


def _check(t: Optional[torch.Tensor], name: str, dtype, device_type: str, numel: Optional[int] = None,
           optional: bool = False):
    if t is None:
        if optional:
            return
        raise ValueError(f"{name} is required")
    if t.dtype not in (dtype if isinstance(dtype, tuple) else (dtype,)):
        raise TypeError(f"{name}: expected {dtype}, got {t.dtype}")
    if t.device.type != device_type:
        raise ValueError(f"{name}: expected a {device_type} tensor, got {t.device}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"{name}: needs at least {numel} elements, has {t.numel()}")


def deinterleave_host_static(delayed: torch.Tensor, grid_out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """cfgms_deinterleave_host_static: CPU int32 [n][T][S] -> CPU int32 [n][T-S+1][S] without a Context and
    without any device allocation by the library — for processes that cannot call cudaMalloc once they are
    serving (all free HBM already belongs to the engine's cache pool, or an allocation's device-wide
    synchronisation would stall the decode streams).  The staging is a fixed CFGMS_STATIC_SCRATCH_BYTES array
    inside the library: a larger request raises CfgmsError with status CFGMS_ERR_LIMIT (split the batch); calls
    share that array, so do not run two of them concurrently on one GPU.  Make the first call on a device at
    start-up (it does a one-time address lookup).  `grid_out` is allocated here on the HOST when not given."""
    _check(delayed, "delayed", torch.int32, "cpu")
    if delayed.dim() != 3:
        raise ValueError("delayed must be [n][T][S]")
    n, T, S = (int(x) for x in delayed.shape)
    if grid_out is None:
        grid_out = torch.empty((n, max(T - S + 1, 0), S), dtype=torch.int32)
    _check(grid_out, "grid_out", torch.int32, "cpu", n * max(T - S + 1, 0) * S)
    sp = stream.cuda_stream if stream is not None else (torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0)
    rc = _lib().cfgms_deinterleave_host_static(delayed.data_ptr(), n, T, S, grid_out.data_ptr(), sp)
    if rc != 0:
        raise CfgmsError(rc, "cfgms_deinterleave_host_static")
    return grid_out


class Context:
    """cfgms_create / cfgms_destroy.  `heads` (bf16 [S][V][d], cuda) is borrowed: kept alive here."""

    def __init__(self, heads: torch.Tensor, embeds: torch.Tensor, max_rows: int = 1024,
                 pad_token: Optional[int] = None, row_tile: int = 0, no_candidates: bool = False,
                 cta_pair: Optional[bool] = None, no_overlap: bool = False, max_stages: int = 0,
                 force_overlap: bool = False, stream_base: int = 0, stream_stride: int = 0,
                 no_pdl_finalize: bool = False, global_streams: int = 0, probe: int = 0,
                 no_split_k: bool = False):
        _check(heads, "heads", torch.bfloat16, "cuda")
        _check(embeds, "embeds", torch.bfloat16, "cuda")
        if heads.dim() != 3 or embeds.dim() != 2 or embeds.shape != (heads.shape[0], heads.shape[2]):
            raise ValueError("heads must be [S][V][d] and embeds [S][d]")
        self.S, self.V, self.d = (int(x) for x in heads.shape)
        self._heads = heads
        cfg = cfgms_config()
        cfg.max_rows = int(max_rows)
        cfg.row_tile = int(row_tile)
        cfg.max_stages = int(max_stages)
        cfg.stream_base, cfg.stream_stride = int(stream_base), int(stream_stride)   # stream-sharded heads
        cfg.global_streams = int(global_streams)
        if pad_token is not None:
            cfg.pad_token = int(pad_token)
            cfg.flags |= CFGMS_CFG_PAD_TOKEN
        if no_candidates:
            cfg.flags |= CFGMS_CFG_NO_CANDIDATES
        if cta_pair is not None:   # tuning: force the one-CTA or the CTA-pair head GEMM
            cfg.flags |= CFGMS_CFG_CTA_PAIR if cta_pair else CFGMS_CFG_SINGLE_CTA
        if no_overlap:             # tuning: finalize strictly after the head GEMM
            cfg.flags |= CFGMS_CFG_NO_OVERLAP
        elif force_overlap:        # tuning: overlap even for a one-wave GEMM
            cfg.flags |= CFGMS_CFG_OVERLAP
        if no_pdl_finalize:        # tuning: finalize kernel always as an ordinary stream-ordered launch
            cfg.flags |= CFGMS_CFG_NO_PDL_FINALIZE
        if no_split_k:             # tuning: never run a one-wave head GEMM as split-K clusters
            cfg.flags |= CFGMS_CFG_NO_SPLIT_K
        # measurement probes (bench.py --probes): two flag bits only the probe build of the library knows (use_library);
        # the product library answers them with CFGMS_ERR_ARG
        cfg.flags |= int(probe) & 0x300
        self.pad_token = self.V if pad_token is None else int(pad_token)
        h = C.c_void_p()
        with torch.cuda.device(heads.device):
            rc = _lib().cfgms_create(C.byref(h), heads.data_ptr(), embeds.data_ptr(), self.S, self.d, self.V,
                                     C.byref(cfg))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_create")
        self._h = h
        self.device = heads.device

    def close(self):
        if getattr(self, "_h", None):
            _lib().cfgms_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _args(self, hidden, pair_map, w, temp, top_k, seed, step, tokens_out, req_id, n_frames, delayed,
              logits_out, dev: str, force_token=None, frame_out=None, frame_index_out=None, eos_token=-1,
              step_next_out=None, n_frames_next_out=None, done_out=None, phase=None, phase_pos=None,
              phase_next_out=None, phase_pos_next_out=None, modality_out=None) -> cfgms_step_args:
        R = int(hidden.shape[0])
        _check(hidden, "hidden", (torch.bfloat16, torch.float32), dev, R * self.d)
        if hidden.dim() != 2 or hidden.shape[1] != self.d:
            raise ValueError("hidden must be [R][d]")
        _check(pair_map, "pair_map", torch.int32, dev, R)
        _check(w, "w", torch.float32, dev, R)
        _check(temp, "temp", torch.float32, dev, R)
        _check(top_k, "top_k", torch.int32, dev, R)
        _check(step, "step", torch.int32, dev, R)
        _check(req_id, "req_id", torch.int32, dev, R, optional=True)
        _check(n_frames, "n_frames", torch.int32, dev, R, optional=True)
        _check(tokens_out, "tokens_out", torch.int32, dev, R * self.S)
        _check(delayed, "delayed", torch.int32, "cuda", optional=True)
        _check(logits_out, "logits_out", torch.float32, "cuda", R * self.S * self.V, optional=True)
        a = cfgms_step_args()
        a.hidden = hidden.data_ptr()
        a.hidden_dtype = CFGMS_F32 if hidden.dtype == torch.float32 else CFGMS_BF16
        a.R = R
        a.pair_map, a.w, a.temp, a.top_k = pair_map.data_ptr(), w.data_ptr(), temp.data_ptr(), top_k.data_ptr()
        a.seed = int(seed) & 0xFFFFFFFFFFFFFFFF
        a.step = step.data_ptr()
        a.req_id, a.n_frames = _ptr(req_id), _ptr(n_frames)
        a.tokens_out = tokens_out.data_ptr()
        if delayed is not None:
            if delayed.dim() != 3 or delayed.shape[0] < R or delayed.shape[2] != self.S:
                raise ValueError("delayed must be [>=R][T_cap][S]")
            a.delayed = delayed.data_ptr()
            a.T_cap = int(delayed.shape[1])
        a.logits_out = _ptr(logits_out)
        _check(force_token, "force_token", torch.int32, dev, R * self.S, optional=True)
        _check(frame_out, "frame_out", torch.int32, dev, R * self.S, optional=True)
        _check(frame_index_out, "frame_index_out", torch.int32, dev, R, optional=True)
        a.force_token, a.frame_out, a.frame_index_out = _ptr(force_token), _ptr(frame_out), _ptr(frame_index_out)
        for t, name in ((step_next_out, "step_next_out"), (n_frames_next_out, "n_frames_next_out"), (done_out, "done_out")):
            _check(t, name, torch.int32, "cuda", R, optional=True)
        a.eos_token = int(eos_token)
        a.step_next_out, a.n_frames_next_out, a.done_out = _ptr(step_next_out), _ptr(n_frames_next_out), _ptr(done_out)
        for t, name in ((phase, "phase"), (phase_pos, "phase_pos")):          # inputs: where the step's inputs live
            _check(t, name, torch.int32, dev, R, optional=True)
        for t, name in ((phase_next_out, "phase_next_out"), (phase_pos_next_out, "phase_pos_next_out"), (modality_out, "modality_out")):
            _check(t, name, torch.int32, "cuda", R, optional=True)           # request state stays in HBM
        a.phase, a.phase_pos = _ptr(phase), _ptr(phase_pos)
        a.phase_next_out, a.phase_pos_next_out, a.modality_out = _ptr(phase_next_out), _ptr(phase_pos_next_out), _ptr(modality_out)
        return a

    def step(self, hidden, pair_map, w, temp, top_k, seed, step, tokens_out, req_id=None, n_frames=None,
             delayed=None, logits_out=None, stream=None, force_token=None, frame_out=None,
             frame_index_out=None, eos_token=-1, step_next_out=None, n_frames_next_out=None, done_out=None,
             phase=None, phase_pos=None, phase_next_out=None, phase_pos_next_out=None, modality_out=None) -> None:
        """cfgms_step: device tensors, enqueue only."""
        a = self._args(hidden, pair_map, w, temp, top_k, seed, step, tokens_out, req_id, n_frames, delayed,
                       logits_out, "cuda", force_token, frame_out, frame_index_out, eos_token, step_next_out,
                       n_frames_next_out, done_out, phase, phase_pos, phase_next_out, phase_pos_next_out, modality_out)
        rc = _lib().cfgms_step(self._h, C.byref(a), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_step")

    def step_host(self, hidden, pair_map, w, temp, top_k, seed, step, tokens_out, req_id=None, n_frames=None,
                  delayed=None, logits_out=None, stream=None, force_token=None, frame_out=None,
                  frame_index_out=None, eos_token=-1, step_next_out=None, n_frames_next_out=None, done_out=None,
                  phase=None, phase_pos=None, phase_next_out=None, phase_pos_next_out=None, modality_out=None) -> None:
        """cfgms_step_host: host tensors in (phase / phase_pos included), host tokens out; the request-state
        outputs, `delayed` and `logits_out` are device tensors; synchronises the stream."""
        a = self._args(hidden, pair_map, w, temp, top_k, seed, step, tokens_out, req_id, n_frames, delayed,
                       logits_out, "cpu", force_token, frame_out, frame_index_out, eos_token, step_next_out,
                       n_frames_next_out, done_out, phase, phase_pos, phase_next_out, phase_pos_next_out, modality_out)
        rc = _lib().cfgms_step_host(self._h, C.byref(a), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_step_host")

    def set_logit_bias(self, bias: Optional[torch.Tensor], stream=None) -> None:
        """cfgms_set_logit_bias: fp32 [S][V] additive vocabulary mask / bias (cuda), or None to clear."""
        _check(bias, "bias", torch.float32, "cuda", self.S * self.V, optional=True)
        rc = _lib().cfgms_set_logit_bias(self._h, _ptr(bias), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_set_logit_bias")

    def set_stream_vocab_sizes(self, sizes, extra_bias: Optional[torch.Tensor] = None, stream=None) -> None:
        """cfgms_set_stream_vocab_sizes: ragged per-stream vocabularies (e.g. one SSL stream + eight codec streams
        of different sizes) on the uniform [S][V][d] layout: stream i only ever samples tokens
        < sizes[i]; `extra_bias` (fp32 [S][V], cuda) is added as well.  The mask is built and folded by the library."""
        sizes = [int(x) for x in sizes]
        if len(sizes) != self.S:
            raise ValueError("sizes must hold S values")
        _check(extra_bias, "extra_bias", torch.float32, "cuda", self.S * self.V, optional=True)
        arr = (C.c_int32 * self.S)(*sizes)
        rc = _lib().cfgms_set_stream_vocab_sizes(self._h, arr, _ptr(extra_bias), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_set_stream_vocab_sizes")

    # ---- stream-sharded heads: the token exchange (cfgms_exchange_*) ----
    def exchange_create(self, world: int, rank: int):
        """-> (64-byte CUDA IPC handle, device address) of this rank's exchange block."""
        handle = (C.c_ubyte * 64)()
        base = C.c_void_p()
        rc = _lib().cfgms_exchange_create(self._h, int(world), int(rank), handle, C.byref(base))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_exchange_create")
        self._xchg = (int(world), int(rank))
        return bytes(handle), int(base.value)

    def exchange_connect(self, peer_bases) -> None:
        """peer_bases: the ranks' block addresses as valid in this process (same-process peers), one per rank."""
        world = getattr(self, "_xchg", (None, None))[0]
        if world is None:
            raise ValueError("exchange_connect before exchange_create")
        if len(peer_bases) != world:       # the library reads exactly `world` entries
            raise ValueError(f"peer_bases needs one entry per rank: world = {world}, got {len(peer_bases)}")
        arr = (C.c_void_p * len(peer_bases))(*[int(b) if b else None for b in peer_bases])
        rc = _lib().cfgms_exchange_connect(self._h, arr)
        if rc != 0:
            raise CfgmsError(rc, "cfgms_exchange_connect")

    def exchange_connect_ipc(self, handles) -> None:
        """handles: every rank's 64-byte IPC handle, in rank order."""
        blob = b"".join(bytes(h) for h in handles)
        if len(blob) != 64 * len(handles):
            raise ValueError("every handle must be 64 bytes")
        world = getattr(self, "_xchg", (None, None))[0]
        if world is None:
            raise ValueError("exchange_connect_ipc before exchange_create")
        if len(handles) != world:          # the library reads world x 64 bytes
            raise ValueError(f"handles needs one entry per rank: world = {world}, got {len(handles)}")
        rc = _lib().cfgms_exchange_connect_ipc(self._h, blob)
        if rc != 0:
            raise CfgmsError(rc, "cfgms_exchange_connect_ipc")

    def exchange_wait(self, R: int, stream=None) -> None:
        rc = _lib().cfgms_exchange_wait(self._h, int(R), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_exchange_wait")

    def exchange_tokens(self, R: int, S_global: int) -> torch.Tensor:
        """This rank's gather buffer as an int32 [R][S_global] tensor view (no copy; owned by the context)."""
        p = C.c_void_p()
        rc = _lib().cfgms_exchange_tokens(self._h, C.byref(p))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_exchange_tokens")
        iface = {"shape": (int(R), int(S_global)), "typestr": "<i4", "data": (int(p.value), False), "version": 3,
                 "strides": None}
        holder = type("_CfgmsView", (), {"__cuda_array_interface__": iface})()
        t = torch.as_tensor(holder, device=self.device)
        t._cfgms_owner = self          # keep the context (and its block) alive
        return t

    def set_phase_table(self, V_text: int, bridge_tokens=()) -> None:
        """cfgms_set_phase_table: text region [0, V_text) of stream 0 and the transition phase's bridging tokens."""
        br = [int(x) for x in bridge_tokens]
        arr = (C.c_int32 * max(len(br), 1))(*br)
        rc = _lib().cfgms_set_phase_table(self._h, int(V_text), arr, len(br))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_set_phase_table")

    def feedback(self, tokens: torch.Tensor, emb: torch.Tensor, x_out: Optional[torch.Tensor] = None,
                 stream=None) -> torch.Tensor:
        """cfgms_feedback: tokens int32 [R][S], emb bf16 [S][V_e][d] -> x bf16 [R][d] (all cuda)."""
        if tokens.dim() != 2 or tokens.shape[1] != self.S or emb.dim() != 3 or emb.shape[0] != self.S \
                or emb.shape[2] != self.d:
            raise ValueError("tokens must be [R][S] and emb [S][V_e][d]")
        R, V_e = int(tokens.shape[0]), int(emb.shape[1])
        _check(tokens, "tokens", torch.int32, "cuda", R * self.S)
        _check(emb, "emb", torch.bfloat16, "cuda", self.S * V_e * self.d)
        if x_out is None:
            x_out = torch.empty((R, self.d), dtype=torch.bfloat16, device=tokens.device)
        _check(x_out, "x_out", torch.bfloat16, "cuda", R * self.d)
        rc = _lib().cfgms_feedback(self._h, tokens.data_ptr(), emb.data_ptr(), V_e, R, x_out.data_ptr(),
                                   _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_feedback")
        return x_out

    def deinterleave(self, delayed: torch.Tensor, grid_out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """cfgms_deinterleave(_host): [n][T][S] int32 -> [n][T-S+1][S]; host path if `delayed` is on the CPU."""
        dev = delayed.device.type
        _check(delayed, "delayed", torch.int32, dev)
        if delayed.dim() != 3:
            raise ValueError("delayed must be [n][T][S]")
        n, T, S = (int(x) for x in delayed.shape)
        if grid_out is None:
            grid_out = torch.empty((n, max(T - S + 1, 0), S), dtype=torch.int32, device=delayed.device)
        _check(grid_out, "grid_out", torch.int32, dev, n * max(T - S + 1, 0) * S)
        fn = _lib().cfgms_deinterleave if dev == "cuda" else _lib().cfgms_deinterleave_host
        rc = fn(self._h, delayed.data_ptr(), n, T, S, grid_out.data_ptr(), _stream_ptr(stream))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_deinterleave")
        return grid_out

    def last_device_error(self):
        """-> (status, row); clears the sticky word; synchronises."""
        row = C.c_int32(-1)
        rc = _lib().cfgms_last_device_error(self._h, C.byref(row))
        return rc, int(row.value)

    def profile_enable(self, on: bool) -> None:
        rc = _lib().cfgms_profile_enable(self._h, int(bool(on)))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_profile_enable")

    def profile_read(self):
        """-> (head-GEMM ms, finalize ms, steps) summed since the last read; synchronises."""
        g, f, n = C.c_double(), C.c_double(), C.c_int64()
        rc = _lib().cfgms_profile_read(self._h, C.byref(g), C.byref(f), C.byref(n))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_profile_read")
        return float(g.value), float(f.value), int(n.value)

    def overlap_stats(self) -> int:
        """-> cells that reached their readiness check while the head GEMM was still producing their
        group, since the last call (evidence of the K1/K2 overlap); synchronises."""
        w = C.c_int64()
        rc = _lib().cfgms_overlap_stats(self._h, C.byref(w))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_overlap_stats")
        return int(w.value)

    def info(self) -> dict:
        inf = cfgms_info()
        rc = _lib().cfgms_get_info(self._h, C.byref(inf))
        if rc != 0:
            raise CfgmsError(rc, "cfgms_get_info")
        return {name: int(getattr(inf, name)) for name, _ in cfgms_info._fields_}
