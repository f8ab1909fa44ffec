"""ctypes binding of libasynclane.so -- argument marshalling only.

Same names as the C ABI (include/asynclane.h).  Arguments are torch CUDA tensors (used purely as
device memory) or raw ints; every step of the path runs in the library's kernels.  There is no CPU
fallback: loading fails loudly if the library is missing, and al_create fails without a B200.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

AL_OK, AL_ERR_INVALID_ARG, AL_ERR_UNSUPPORTED, AL_ERR_WORKSPACE, AL_ERR_CUDA = range(5)
AL_F32, AL_BF16 = 0, 1
AL_LANE_FLAG_REFINE = 1
AL_SELECT_FORCE_TOP1 = 1

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libasynclane.so")

EXPORTS = [
    "al_create", "al_destroy", "al_last_error", "al_version", "al_sm_count",
    "al_lane_attention_workspace_bytes", "al_lane_attention", "al_lane_plan", "al_lane_attention_planned",
    "al_kv_refresh", "al_refresh_forward", "al_lane_status", "al_scheduler_run", "al_stub_model_fn",
    "al_confidence_select_workspace_bytes", "al_confidence_select", "al_lm_head_confidence_workspace_bytes",
    "al_lm_head_confidence", "al_lm_head_confidence_static_max_bytes", "al_lm_head_confidence_static",
    "al_validate_lanes", "al_validate_refresh",
    "al_selftest_umma", "al_lane_step_host", "al_lane_step_host_arena_bytes", "al_lane_step_host_traffic",
    "al_launch_count",
]


class AlError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"asynclane status {status}: {message}")
        self.status = status


class al_attn_shape(ctypes.Structure):
    _fields_ = [("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("dtype", ctypes.c_int32), ("cache_rows", ctypes.c_int64), ("scale", ctypes.c_float),
                ("reserved", ctypes.c_int32)]


class al_host_step(ctypes.Structure):
    """Mirror of al_host_step (include/asynclane.h): HOST pointers of one step's inputs and results."""
    _fields_ = [("q", ctypes.c_void_p), ("k_new", ctypes.c_void_p), ("v_new", ctypes.c_void_p),
                ("lanes", ctypes.c_void_p), ("n_lanes", ctypes.c_int32), ("total_q_rows", ctypes.c_int32),
                ("max_prefix_len", ctypes.c_int32),
                ("k_src", ctypes.c_void_p), ("v_src", ctypes.c_void_p), ("pos", ctypes.c_void_p),
                ("n_pos", ctypes.c_int32), ("refresh_base_row", ctypes.c_int32),
                ("logits", ctypes.c_void_p), ("n_rows", ctypes.c_int32), ("vocab", ctypes.c_int32),
                ("tokens_in", ctypes.c_void_p), ("mask_id", ctypes.c_int32), ("eos_id", ctypes.c_int32),
                ("threshold", ctypes.c_float), ("select_flags", ctypes.c_int32),
                ("out", ctypes.c_void_p), ("conf", ctypes.c_void_p), ("argmax", ctypes.c_void_p),
                ("commit", ctypes.c_void_p), ("tokens_out", ctypes.c_void_p),
                ("n_layers", ctypes.c_int32), ("reserved", ctypes.c_int32), ("cache_layer_stride", ctypes.c_int64)]


class al_sched_config(ctypes.Structure):
    """Mirror of al_sched_config (include/asynclane.h): Algorithm 1's parameters; the id lists are HOST arrays."""
    _fields_ = [("prompt_len", ctypes.c_int32), ("gen_len", ctypes.c_int32), ("block_size", ctypes.c_int32),
                ("lookahead", ctypes.c_int32), ("vocab", ctypes.c_int32), ("mask_id", ctypes.c_int32),
                ("eos_id", ctypes.c_int32), ("tau", ctypes.c_float), ("tau_future", ctypes.c_float),
                ("rho_min", ctypes.c_float), ("t_min", ctypes.c_int32), ("max_lane_steps", ctypes.c_int32),
                ("max_iterations", ctypes.c_int32), ("refresh_period", ctypes.c_int32),
                ("refresh_margin", ctypes.c_int32), ("delimiter_ids", ctypes.c_void_p), ("n_delimiters", ctypes.c_int32),
                ("no_fork_prev_ids", ctypes.c_void_p), ("n_no_fork_prev", ctypes.c_int32)]


class al_sched_lane(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("role", "start", "len", "steps", "parent", "ref_child", "gen_child",
                                              "successor", "state", "valid_prefix", "split_point", "n_masked")]


class al_sched_stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("iterations", "model_calls", "lane_forwards", "forks", "successors",
                                              "refreshes", "stopped_frontiers", "rows_forwarded", "tokens_committed",
                                              "tokens_drafted", "refreshed_rows_last", "reserved")]


class al_stub_model(ctypes.Structure):
    _fields_ = [("base_dev", ctypes.c_void_p), ("target_dev", ctypes.c_void_p), ("gain", ctypes.c_float),
                ("vocab", ctypes.c_int32)]


class al_sched_device_state(ctypes.Structure):
    _fields_ = [("shape", al_attn_shape), ("k_cache", ctypes.c_void_p), ("v_cache", ctypes.c_void_p),
                ("k_src", ctypes.c_void_p), ("v_src", ctypes.c_void_p), ("q", ctypes.c_void_p),
                ("k_new", ctypes.c_void_p), ("v_new", ctypes.c_void_p), ("out", ctypes.c_void_p),
                ("max_rows", ctypes.c_int32)]


AL_MODEL_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
                               ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)

_lib: Optional[ctypes.CDLL] = None


def load_library(build_if_missing: bool = True) -> ctypes.CDLL:
    """dlopen libasynclane.so (building it in-tree first if absent) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise FileNotFoundError(f"{LIB_PATH} missing: run `python -m paper_2606_08411_b200.build`")
        from . import build as _build
        _build.build()
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, f32, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_size_t
    shp = ctypes.POINTER(al_attn_shape)
    lib.al_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int]
    lib.al_destroy.argtypes = [vp]
    lib.al_last_error.restype = ctypes.c_char_p
    lib.al_version.restype = ctypes.c_char_p
    lib.al_sm_count.argtypes = [vp]
    lib.al_sm_count.restype = i32
    lib.al_lane_attention_workspace_bytes.argtypes = [shp, i32, i32, i32]
    lib.al_lane_attention_workspace_bytes.restype = sz
    lib.al_lane_attention.argtypes = [vp, shp, vp, vp, vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, sz, vp]
    lib.al_lane_attention_planned.argtypes = lib.al_lane_attention.argtypes
    lib.al_refresh_forward.argtypes = lib.al_lane_attention.argtypes
    lib.al_lane_plan.argtypes = [vp, shp, vp, i32, i32, i32, vp, sz, vp]
    lib.al_kv_refresh.argtypes = [vp, shp, vp, vp, vp, vp, vp, i32, i32, i32, i64, i64, vp]
    lib.al_confidence_select_workspace_bytes.argtypes = [i32, i32]
    lib.al_confidence_select_workspace_bytes.restype = sz
    lib.al_confidence_select.argtypes = [vp, vp, i32, i32, i32, i64, vp, i32, i32, f32, vp, i32, i32,
                                         vp, vp, vp, vp, vp, sz, vp]
    lib.al_lm_head_confidence_workspace_bytes.argtypes = [i32, i32]
    lib.al_lm_head_confidence_workspace_bytes.restype = sz
    lib.al_lm_head_confidence.argtypes = [vp, vp, vp, i32, i32, i32, vp, i32, i32, f32, vp, i32, i32, vp, vp, vp, vp, vp,
                                          sz, vp]
    lib.al_lm_head_confidence_static_max_bytes.argtypes = []
    lib.al_lm_head_confidence_static_max_bytes.restype = sz
    lib.al_lm_head_confidence_static.argtypes = [vp, vp, vp, i32, i32, i32, vp, i32, i32, f32, vp, i32, i32, vp, vp, vp, vp,
                                                 vp]
    lib.al_lane_status.argtypes = [vp, vp, i32, i32, vp, vp, vp, i32, i32, f32, vp, i32, vp, i32, vp, vp, vp, vp]
    lib.al_scheduler_run.argtypes = [vp, ctypes.POINTER(al_sched_config), vp, vp, ctypes.POINTER(al_sched_device_state),
                                     vp, vp, vp, ctypes.POINTER(i32), ctypes.POINTER(al_sched_lane), i32,
                                     ctypes.POINTER(i32), ctypes.POINTER(al_sched_stats), vp]
    lib.al_validate_lanes.argtypes = [vp, shp, vp, i32, i32]
    lib.al_validate_refresh.argtypes = [vp, shp, vp, i32, i32]
    lib.al_selftest_umma.argtypes = [vp, vp, vp, vp, f32, vp, vp, vp]
    hsp = ctypes.POINTER(al_host_step)
    lib.al_lane_step_host_arena_bytes.argtypes = [shp, hsp]
    lib.al_lane_step_host_arena_bytes.restype = sz
    lib.al_lane_step_host.argtypes = [vp, shp, hsp, vp, vp, vp, sz, vp]
    lib.al_lane_step_host_traffic.argtypes = [shp, hsp, ctypes.POINTER(ctypes.c_uint64),
                                              ctypes.POINTER(ctypes.c_uint64)]
    lib.al_lane_step_host_traffic.restype = None
    lib.al_launch_count.argtypes = [vp]
    lib.al_launch_count.restype = ctypes.c_uint64
    for name in EXPORTS:
        fn = getattr(lib, name)
        if name not in ("al_last_error", "al_version", "al_sm_count", "al_lane_attention_workspace_bytes",
                        "al_confidence_select_workspace_bytes", "al_lane_step_host_arena_bytes",
                        "al_lm_head_confidence_workspace_bytes", "al_lm_head_confidence_static_max_bytes",
                        "al_lane_step_host_traffic", "al_launch_count", "al_stub_model_fn"):
            fn.restype = ctypes.c_int
    _lib = lib
    return lib


def _check(status: int) -> None:
    if status != AL_OK:
        raise AlError(status, load_library().al_last_error().decode())


def _ptr(t) -> Optional[int]:
    """Device pointer of a torch CUDA tensor (None passes NULL)."""
    if t is None:
        return None
    if not t.is_cuda:
        raise TypeError("asynclane: expected a CUDA tensor (the library has no CPU path)")
    if not t.is_contiguous():
        raise ValueError("asynclane: tensors must be contiguous")
    return t.data_ptr()


def _dtype_code(t) -> int:
    import torch
    if t.dtype == torch.bfloat16:
        return AL_BF16
    if t.dtype == torch.float32:
        return AL_F32
    raise TypeError(f"asynclane: unsupported dtype {t.dtype}")


def _stream_ptr(stream) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


class Handle:
    """Owns an al_handle; methods carry the names of the C entry points."""

    def __init__(self, device: int = 0):
        self._lib = load_library()
        h = ctypes.c_void_p()
        _check(self._lib.al_create(ctypes.byref(h), device))
        self._h = h
        self.device = device

    def close(self) -> None:
        if getattr(self, "_h", None):
            self._lib.al_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def sm_count(self) -> int:
        return int(self._lib.al_sm_count(self._h))

    @staticmethod
    def make_shape(n_q_heads: int, n_kv_heads: int, head_dim: int, dtype: int, cache_rows: int,
                   scale: float = 0.0) -> al_attn_shape:
        return al_attn_shape(n_q_heads, n_kv_heads, head_dim, dtype, cache_rows, scale, 0)

    def al_lane_attention_workspace_bytes(self, shape: al_attn_shape, n_lanes: int, total_q_rows: int,
                                          max_prefix_len: int) -> int:
        return int(self._lib.al_lane_attention_workspace_bytes(ctypes.byref(shape), n_lanes, total_q_rows,
                                                               max_prefix_len))

    def al_lane_attention(self, shape, q, k_new, v_new, k_cache, v_cache, lanes_dev, n_lanes, total_q_rows,
                          max_prefix_len, out, lse=None, workspace=None, stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_lane_attention(self._h, ctypes.byref(shape), _ptr(q), _ptr(k_new), _ptr(v_new),
                                           _ptr(k_cache), _ptr(v_cache), _ptr(lanes_dev), n_lanes, total_q_rows,
                                           max_prefix_len, _ptr(out), _ptr(lse), _ptr(workspace), ws_bytes,
                                           _stream_ptr(stream)))

    def al_refresh_forward(self, shape, q, k_new, v_new, k_cache, v_cache, lanes_dev, n_lanes, total_q_rows,
                           max_prefix_len, out, lse=None, workspace=None, stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_refresh_forward(self._h, ctypes.byref(shape), _ptr(q), _ptr(k_new), _ptr(v_new),
                                            _ptr(k_cache), _ptr(v_cache), _ptr(lanes_dev), n_lanes, total_q_rows,
                                            max_prefix_len, _ptr(out), _ptr(lse), _ptr(workspace), ws_bytes,
                                            _stream_ptr(stream)))

    def al_lane_plan(self, shape, lanes_dev, n_lanes, total_q_rows, max_prefix_len, workspace, stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_lane_plan(self._h, ctypes.byref(shape), _ptr(lanes_dev), n_lanes, total_q_rows,
                                      max_prefix_len, _ptr(workspace), ws_bytes, _stream_ptr(stream)))

    def al_lane_attention_planned(self, shape, q, k_new, v_new, k_cache, v_cache, lanes_dev, n_lanes,
                                  total_q_rows, max_prefix_len, out, lse=None, workspace=None, stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_lane_attention_planned(self._h, ctypes.byref(shape), _ptr(q), _ptr(k_new), _ptr(v_new),
                                                   _ptr(k_cache), _ptr(v_cache), _ptr(lanes_dev), n_lanes,
                                                   total_q_rows, max_prefix_len, _ptr(out), _ptr(lse),
                                                   _ptr(workspace), ws_bytes, _stream_ptr(stream)))

    def al_kv_refresh(self, shape, k_cache, v_cache, k_src, v_src, pos_dev, n_pos, kv_base_row=0, n_layers=1,
                      layer_stride_cache=0, layer_stride_src=0, stream=None) -> None:
        _check(self._lib.al_kv_refresh(self._h, ctypes.byref(shape), _ptr(k_cache), _ptr(v_cache), _ptr(k_src),
                                       _ptr(v_src), _ptr(pos_dev), n_pos, kv_base_row, n_layers,
                                       layer_stride_cache, layer_stride_src, _stream_ptr(stream)))

    def al_confidence_select_workspace_bytes(self, n_rows: int, vocab: int) -> int:
        return int(self._lib.al_confidence_select_workspace_bytes(n_rows, vocab))

    def al_confidence_select(self, logits, n_rows, vocab, row_stride, tokens_in, mask_id, eos_id, threshold,
                             lanes_dev, n_lanes, flags, conf_out, argmax_out, commit_out, tokens_out,
                             workspace, stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_confidence_select(self._h, _ptr(logits), _dtype_code(logits), n_rows, vocab,
                                              row_stride, _ptr(tokens_in), mask_id, eos_id, threshold,
                                              _ptr(lanes_dev), n_lanes, flags, _ptr(conf_out), _ptr(argmax_out),
                                              _ptr(commit_out), _ptr(tokens_out), _ptr(workspace), ws_bytes,
                                              _stream_ptr(stream)))

    @property
    def al_launch_count(self) -> int:
        return int(self._lib.al_launch_count(self._h))

    def al_lane_step_host_arena_bytes(self, shape: al_attn_shape, step: al_host_step) -> int:
        return int(self._lib.al_lane_step_host_arena_bytes(ctypes.byref(shape), ctypes.byref(step)))

    def al_lane_step_host_traffic(self, shape: al_attn_shape, step: al_host_step):
        a, b = ctypes.c_uint64(0), ctypes.c_uint64(0)
        self._lib.al_lane_step_host_traffic(ctypes.byref(shape), ctypes.byref(step), ctypes.byref(a), ctypes.byref(b))
        return int(a.value), int(b.value)

    def al_lane_step_host(self, shape, step: al_host_step, k_cache, v_cache, arena, stream=None) -> None:
        """`step` holds HOST pointers (pinned torch tensors' data_ptr()); caches/arena are CUDA tensors."""
        _check(self._lib.al_lane_step_host(self._h, ctypes.byref(shape), ctypes.byref(step), _ptr(k_cache),
                                           _ptr(v_cache), _ptr(arena), arena.numel() * arena.element_size(),
                                           _stream_ptr(stream)))

    def al_validate_lanes(self, shape, lanes_dev, n_lanes, total_q_rows) -> None:
        _check(self._lib.al_validate_lanes(self._h, ctypes.byref(shape), _ptr(lanes_dev), n_lanes, total_q_rows))

    def al_lm_head_confidence_workspace_bytes(self, n_rows: int, vocab: int) -> int:
        return int(self._lib.al_lm_head_confidence_workspace_bytes(n_rows, vocab))

    def al_lm_head_confidence(self, hidden, weight, n_rows, vocab, hidden_dim, tokens_in, mask_id, eos_id, threshold,
                              lanes_dev, n_lanes, flags, conf_out, argmax_out, commit_out, tokens_out, workspace,
                              stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        _check(self._lib.al_lm_head_confidence(self._h, _ptr(hidden), _ptr(weight), n_rows, vocab, hidden_dim,
                                               _ptr(tokens_in), mask_id, eos_id, threshold, _ptr(lanes_dev), n_lanes,
                                               flags, _ptr(conf_out), _ptr(argmax_out), _ptr(commit_out),
                                               _ptr(tokens_out), _ptr(workspace), ws_bytes, _stream_ptr(stream)))

    def al_lm_head_confidence_static_max_bytes(self) -> int:
        return int(self._lib.al_lm_head_confidence_static_max_bytes())

    def al_lm_head_confidence_static(self, hidden, weight, n_rows, vocab, hidden_dim, tokens_in, mask_id, eos_id,
                                     threshold, lanes_dev, n_lanes, flags, conf_out, argmax_out, commit_out, tokens_out,
                                     stream=None) -> None:
        """al_lm_head_confidence without a workspace: the partials live in the library's static device array."""
        _check(self._lib.al_lm_head_confidence_static(self._h, _ptr(hidden), _ptr(weight), n_rows, vocab, hidden_dim,
                                                      _ptr(tokens_in), mask_id, eos_id, threshold, _ptr(lanes_dev),
                                                      n_lanes, flags, _ptr(conf_out), _ptr(argmax_out),
                                                      _ptr(commit_out), _ptr(tokens_out), _stream_ptr(stream)))

    def al_lane_status(self, lanes_dev, n_lanes, n_rows, tokens_in, conf, argmax, mask_id, eos_id, tau_future,
                       delimiter_ids, no_fork_prev_ids, commit_io, tokens_io, status_out, stream=None) -> None:
        """status_out: int32 CUDA tensor [n_lanes, 8] (al_lane_status_rec)."""
        nd = 0 if delimiter_ids is None else int(delimiter_ids.numel())
        nn = 0 if no_fork_prev_ids is None else int(no_fork_prev_ids.numel())
        _check(self._lib.al_lane_status(self._h, _ptr(lanes_dev), n_lanes, n_rows, _ptr(tokens_in), _ptr(conf),
                                        _ptr(argmax), mask_id, eos_id, tau_future, _ptr(delimiter_ids), nd,
                                        _ptr(no_fork_prev_ids), nn, _ptr(commit_io), _ptr(tokens_io),
                                        _ptr(status_out), _stream_ptr(stream)))

    def al_scheduler_run(self, config: al_sched_config, model_fn, model_user, device_state, prompt_host, x_host,
                         output_host, tree, stream=None):
        """model_fn: a C function pointer (the library's al_stub_model_fn, or an AL_MODEL_FN wrapping a Python
        callable); model_user: ctypes pointer/int passed through; prompt/x/output: int32 numpy arrays (host);
        tree: ctypes array of al_sched_lane.  Returns (n_output, n_tree, al_sched_stats)."""
        n_out, n_tree, stats = ctypes.c_int32(0), ctypes.c_int32(0), al_sched_stats()
        ds = None if device_state is None else ctypes.byref(device_state)
        _check(self._lib.al_scheduler_run(self._h, ctypes.byref(config), ctypes.cast(model_fn, ctypes.c_void_p),
                                          model_user, ds, prompt_host.ctypes.data, x_host.ctypes.data,
                                          output_host.ctypes.data, ctypes.byref(n_out), tree, len(tree),
                                          ctypes.byref(n_tree), ctypes.byref(stats), _stream_ptr(stream)))
        return int(n_out.value), int(n_tree.value), stats

    def al_validate_refresh(self, shape, pos_dev, n_pos, kv_base_row=0) -> None:
        _check(self._lib.al_validate_refresh(self._h, ctypes.byref(shape), _ptr(pos_dev), n_pos, kv_base_row))

    def al_selftest_umma(self, a, b, v, p_scale, s_out, o_out, stream=None) -> None:
        _check(self._lib.al_selftest_umma(self._h, _ptr(a), _ptr(b), _ptr(v), p_scale, _ptr(s_out), _ptr(o_out),
                                          _stream_ptr(stream)))
