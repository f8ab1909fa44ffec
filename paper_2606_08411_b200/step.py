"""Device-resident buffers for one lane-batched denoising step and the three C-ABI calls that make
up the hot path: per layer al_lane_attention, then al_kv_refresh (all layers in one
launch), then al_confidence_select.  Only marshalling and buffer ownership live here; torch is used
for device memory, streams and CUDA graphs.
"""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import binding as B
from .workloads import LaneStepWorkload, bf16_bits


def to_device(x: np.ndarray, dtype: str, device) -> torch.Tensor:
    """float32 array whose values are representable in `dtype` -> device tensor of that dtype."""
    if dtype == "bf16":
        bits = torch.from_numpy(bf16_bits(x).view(np.int16).reshape(x.shape))
        return bits.to(device).view(torch.bfloat16)
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(device)


def to_host_pinned(x: np.ndarray, dtype: str) -> torch.Tensor:
    if dtype == "bf16":
        t = torch.from_numpy(bf16_bits(x).view(np.int16).reshape(x.shape)).view(torch.bfloat16)
    else:
        t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32))
    return t.pin_memory()


class LaneStep:
    """One workload resident on the GPU + outputs + workspaces; `run()` enqueues the whole step."""

    def __init__(self, handle: B.Handle, wl: LaneStepWorkload, device="cuda:0", want_lse: bool = True,
                 force_top1: bool = False):
        self.h = handle
        self.wl = wl
        dev = torch.device(device)
        self.device = dev
        dt = wl.dtype
        self.code = B.AL_BF16 if dt == "bf16" else B.AL_F32
        self.tdtype = torch.bfloat16 if dt == "bf16" else torch.float32
        self.shape = B.Handle.make_shape(wl.n_q_heads, wl.n_kv_heads, wl.head_dim, self.code, wl.cache_rows)
        self.q = to_device(wl.q, dt, dev)
        self.k_new = to_device(wl.k_new, dt, dev)
        self.v_new = to_device(wl.v_new, dt, dev)
        self.k_cache = to_device(wl.k_cache, dt, dev)
        self.v_cache = to_device(wl.v_cache, dt, dev)
        self.k_src = to_device(wl.k_src, dt, dev)
        self.v_src = to_device(wl.v_src, dt, dev)
        self.logits = to_device(wl.logits, dt, dev)
        self.lanes = torch.from_numpy(np.ascontiguousarray(wl.lanes, dtype=np.int32)).to(dev)
        self.pos = torch.from_numpy(np.ascontiguousarray(wl.refresh_pos, dtype=np.int32)).to(dev)
        self.tokens = torch.from_numpy(np.ascontiguousarray(wl.tokens, dtype=np.int32)).to(dev)
        L, T = wl.n_layers, wl.total_q_rows
        N, V = wl.logits.shape
        self.n_layers, self.T, self.N, self.V = L, T, N, V
        self.out = torch.zeros((L, T, wl.n_q_heads, wl.head_dim), dtype=self.tdtype, device=dev)
        self.lse = torch.zeros((L, T, wl.n_q_heads), dtype=torch.float32, device=dev) if want_lse else None
        self.conf = torch.zeros(N, dtype=torch.float32, device=dev)
        self.argmax = torch.zeros(N, dtype=torch.int32, device=dev)
        self.commit = torch.zeros(N, dtype=torch.uint8, device=dev)
        self.tokens_out = torch.zeros(N, dtype=torch.int32, device=dev)
        self.max_prefix = wl.max_prefix_len
        ws_a = handle.al_lane_attention_workspace_bytes(self.shape, wl.n_lanes, T, self.max_prefix)
        ws_c = handle.al_confidence_select_workspace_bytes(N, V)
        self.ws_attn = torch.empty(max(ws_a, 16), dtype=torch.uint8, device=dev)
        self.ws_conf = torch.empty(max(ws_c, 16), dtype=torch.uint8, device=dev)
        self.flags = B.AL_SELECT_FORCE_TOP1 if force_top1 else 0
        self.gpu_launches_per_step = None   # filled by callers that count (bench)
        # side stream of run(overlap=True); made here (not under a graph capture) and shared by replicas
        self._side = torch.cuda.Stream(device=dev)
        self._fork, self._join = torch.cuda.Event(), torch.cuda.Event()

    def replicate(self) -> "LaneStep":
        """A second instance on DISTINCT device allocations of every streamed buffer (same values):
        bench.py rotates over such copies so that consecutive steps never hit in L2."""
        import copy
        r = copy.copy(self)
        for name in ("q", "k_new", "v_new", "k_cache", "v_cache", "k_src", "v_src", "logits", "out", "lse",
                     "conf", "argmax", "commit", "tokens_out", "ws_attn", "ws_conf"):
            t = getattr(self, name)
            setattr(r, name, None if t is None else t.clone())
        return r

    def streamed_bytes(self) -> int:
        """Device bytes one step streams (inputs + caches + outputs), for sizing the L2 rotation."""
        tot = 0
        for name in ("q", "k_new", "v_new", "k_cache", "v_cache", "k_src", "v_src", "logits", "out"):
            t = getattr(self, name)
            tot += t.numel() * t.element_size()
        return tot

    # -- the three parts ---------------------------------------------------------------------------
    def attention(self, stream=None, layers: Optional[range] = None) -> None:
        """al_lane_plan once (the lanes are those of one scheduler iteration), then one
        al_lane_attention_planned per layer."""
        wl = self.wl
        self.h.al_lane_plan(self.shape, self.lanes, wl.n_lanes, self.T, self.max_prefix, self.ws_attn, stream)
        for l in (range(self.n_layers) if layers is None else layers):
            self.h.al_lane_attention_planned(self.shape, self.q[l], self.k_new[l], self.v_new[l], self.k_cache[l],
                                             self.v_cache[l], self.lanes, wl.n_lanes, self.T, self.max_prefix,
                                             self.out[l], None if self.lse is None else self.lse[l], self.ws_attn,
                                             stream)

    def refresh(self, stream=None) -> None:
        wl = self.wl
        R = int(self.pos.numel())
        per_layer_cache = wl.n_kv_heads * wl.cache_rows * wl.head_dim
        per_layer_src = R * wl.n_kv_heads * wl.head_dim
        self.h.al_kv_refresh(self.shape, self.k_cache, self.v_cache, self.k_src, self.v_src, self.pos, R,
                             wl.refresh_base_row, self.n_layers, per_layer_cache, per_layer_src, stream)

    def confidence(self, stream=None) -> None:
        wl = self.wl
        self.h.al_confidence_select(self.logits, self.N, self.V, self.V, self.tokens, wl.mask_id, wl.eos_id,
                                    float(wl.threshold), self.lanes, wl.n_lanes, self.flags, self.conf,
                                    self.argmax, self.commit, self.tokens_out, self.ws_conf, stream)

    # Above this many logits bytes the confidence kernel saturates HBM on its own (cfg5: 98 % of the copy
    # bandwidth) and a concurrent refresh only disturbs its cluster scheduling (measured: +10 us at cfg5,
    # -3.5 us at cfg2, -3 us at cfg3): the refresh then runs in line.
    OVERLAP_MAX_LOGITS_BYTES = 256 << 20

    def run(self, stream=None, marks=None, overlap: Optional[bool] = None) -> None:
        """The whole hot path once.  Attention reads the cache BEFORE this step's refresh writes it
        (kappa_l is the state the lanes were forked from; refresh is periodic, L176).
        Refresh (writes the cache) and confidence/select (reads the logits) are independent of each
        other: with `overlap` (default: when the logits are small enough for it to pay) the refresh runs
        on a side stream, forked after the attention and joined after the confidence kernel -- plain
        edges when the step is captured into a CUDA graph.
        `marks`: optional 4 timing events recorded before/between/after the three parts (serial order)."""
        s = torch.cuda.current_stream() if stream is None else stream
        if overlap is None:
            overlap = self.logits.numel() * self.logits.element_size() <= self.OVERLAP_MAX_LOGITS_BYTES
        if marks is not None:
            overlap = False
            marks[0].record(s)
        self.attention(stream)
        if marks is not None:
            marks[1].record(s)
        if overlap:
            self._fork.record(s)
            self._side.wait_event(self._fork)
            self.refresh(self._side)
            self._join.record(self._side)
            self.confidence(stream)
            s.wait_event(self._join)
            return
        self.refresh(stream)
        if marks is not None:
            marks[2].record(s)
        self.confidence(stream)
        if marks is not None:
            marks[3].record(s)


class HostStep:
    """Pinned HOST buffers of one workload + the al_host_step struct for al_lane_step_host (the e2e entry):
    every layer's Q/K_new/V_new and refresh rows, the logits and the result buffers.  Marshalling only."""

    def __init__(self, handle: B.Handle, wl: LaneStepWorkload, device="cuda:0", force_top1: bool = False):
        self.h, self.wl = handle, wl
        dev = torch.device(device)
        dt = wl.dtype
        code = B.AL_BF16 if dt == "bf16" else B.AL_F32
        tdt = torch.bfloat16 if dt == "bf16" else torch.float32
        self.shape = B.Handle.make_shape(wl.n_q_heads, wl.n_kv_heads, wl.head_dim, code, wl.cache_rows)
        hs = B.al_host_step()
        self.host = {}

        def pin(name, arr, dtype=None):
            t = to_host_pinned(arr, dtype) if dtype else torch.from_numpy(np.ascontiguousarray(arr)).pin_memory()
            self.host[name] = t
            return t.data_ptr()

        L, T = wl.n_layers, wl.total_q_rows
        hs.q, hs.k_new, hs.v_new = pin("q", wl.q, dt), pin("k_new", wl.k_new, dt), pin("v_new", wl.v_new, dt)
        hs.lanes = pin("lanes", wl.lanes.astype(np.int32))
        hs.n_lanes, hs.total_q_rows, hs.max_prefix_len = wl.n_lanes, T, wl.max_prefix_len
        hs.k_src, hs.v_src = pin("k_src", wl.k_src, dt), pin("v_src", wl.v_src, dt)
        hs.pos = pin("pos", wl.refresh_pos.astype(np.int32))
        hs.n_pos, hs.refresh_base_row = int(wl.refresh_pos.size), wl.refresh_base_row
        hs.logits = pin("logits", wl.logits, dt)
        hs.n_rows, hs.vocab = wl.logits.shape
        hs.tokens_in = pin("tokens", wl.tokens.astype(np.int32))
        hs.mask_id, hs.eos_id, hs.threshold = wl.mask_id, wl.eos_id, float(wl.threshold)
        hs.select_flags = B.AL_SELECT_FORCE_TOP1 if force_top1 else 0
        N = int(hs.n_rows)
        self.out = torch.empty((L, T, wl.n_q_heads, wl.head_dim), dtype=tdt).pin_memory()
        self.conf = torch.empty(N, dtype=torch.float32).pin_memory()
        self.argmax = torch.empty(N, dtype=torch.int32).pin_memory()
        self.commit = torch.empty(N, dtype=torch.uint8).pin_memory()
        self.tokens_out = torch.empty(N, dtype=torch.int32).pin_memory()
        hs.out, hs.conf, hs.argmax = self.out.data_ptr(), self.conf.data_ptr(), self.argmax.data_ptr()
        hs.commit, hs.tokens_out = self.commit.data_ptr(), self.tokens_out.data_ptr()
        hs.n_layers, hs.reserved = L, 0
        hs.cache_layer_stride = wl.n_kv_heads * wl.cache_rows * wl.head_dim
        self.hs = hs
        self.arena = torch.empty(handle.al_lane_step_host_arena_bytes(self.shape, hs) + 256, dtype=torch.uint8,
                                 device=dev)
        self.h2d_bytes, self.d2h_bytes = handle.al_lane_step_host_traffic(self.shape, hs)

    def run(self, k_cache: torch.Tensor, v_cache: torch.Tensor, stream=None) -> None:
        """Enqueues one whole step on `stream`; k_cache/v_cache are the resident device caches [L,Hkv,rows,d]."""
        self.h.al_lane_step_host(self.shape, self.hs, k_cache, v_cache, self.arena, stream)
