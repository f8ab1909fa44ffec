"""CPU oracle for the lane-batched denoising step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` may import this package.  The product (``paper_2606_08411_b200``) never does, and
this package never imports the product's kernels or binding (only the seeded input generator
``paper_2606_08411_b200.workloads`` is shared, and that is used by callers, not here).

The arithmetic lives in ``asynclane_oracle.c`` (plain C, fp64, the paper's definitions written
out; see the citations there).  This file only compiles it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "asynclane_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc -O3 -fopenmp); returns the path of the shared object."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O3", "-fopenmp", "-fno-fast-math", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def lane_attention(q, k_new, v_new, k_cache, v_cache, lanes, scale: Optional[float] = None
                   ) -> Tuple[np.ndarray, np.ndarray]:
    """O-A.  q [T,Hq,d]; k_new,v_new [T,Hkv,d]; caches [Hkv,cache_rows,d]; lanes int32 [n,6].
    Returns (out fp64 [T,Hq,d], lse fp64 [T,Hq]).  scale None => 1/sqrt(d) (reading C2)."""
    q, k_new, v_new, k_cache, v_cache = map(_f32, (q, k_new, v_new, k_cache, v_cache))
    lanes = _i32(lanes).reshape(-1, 6)
    T, Hq, d = q.shape
    Hkv, cache_rows = k_cache.shape[0], k_cache.shape[1]
    assert k_new.shape == (T, Hkv, d) and v_new.shape == (T, Hkv, d) and v_cache.shape == k_cache.shape
    assert Hq % Hkv == 0
    if scale is None:
        scale = 1.0 / np.sqrt(float(d))
    out = np.zeros((T, Hq, d), dtype=np.float64)
    lse = np.zeros((T, Hq), dtype=np.float64)
    _load().oracle_lane_attention(_p(q), _p(k_new), _p(v_new), _p(k_cache), _p(v_cache), _p(lanes),
                                  ctypes.c_int(lanes.shape[0]), ctypes.c_int(Hq), ctypes.c_int(Hkv),
                                  ctypes.c_int(d), ctypes.c_int64(cache_rows), ctypes.c_double(scale),
                                  _p(out), _p(lse))
    return out, lse


def lane_attention_one(q, k_new, v_new, k_cache, v_cache, lane, local_row: int, head: int,
                       scale: Optional[float] = None) -> Tuple[np.ndarray, float]:
    """O-A for one (lane, local row, q-head): the sampled-output form for full-size parity."""
    q, k_new, v_new, k_cache, v_cache = map(_f32, (q, k_new, v_new, k_cache, v_cache))
    lane = _i32(lane).reshape(6)
    T, Hq, d = q.shape
    Hkv, cache_rows = k_cache.shape[0], k_cache.shape[1]
    if scale is None:
        scale = 1.0 / np.sqrt(float(d))
    out = np.zeros(d, dtype=np.float64)
    lse = ctypes.c_double(0.0)
    _load().oracle_lane_attention_one(_p(q), _p(k_new), _p(v_new), _p(k_cache), _p(v_cache), _p(lane),
                                      ctypes.c_int(local_row), ctypes.c_int(head), ctypes.c_int(Hq),
                                      ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int64(cache_rows),
                                      ctypes.c_double(scale), _p(out), ctypes.byref(lse))
    return out, float(lse.value)


def kv_refresh(k_cache: np.ndarray, v_cache: np.ndarray, k_src: np.ndarray, v_src: np.ndarray,
               pos, kv_base_row: int = 0) -> None:
    """O-B, IN PLACE on the given arrays (any fixed-size element type; bytes are copied).
    caches [L,Hkv,cache_rows,d] (or [Hkv,cache_rows,d]); src [L,R,Hkv,d] (or [R,Hkv,d])."""
    for a in (k_cache, v_cache, k_src, v_src):
        assert a.flags["C_CONTIGUOUS"]
    assert k_cache.dtype == k_src.dtype == v_cache.dtype == v_src.dtype
    kc = k_cache if k_cache.ndim == 4 else k_cache[None]
    ks = k_src if k_src.ndim == 4 else k_src[None]
    L, Hkv, cache_rows, d = kc.shape
    pos = _i32(pos)
    R = pos.size
    assert ks.shape == (L, R, Hkv, d), (ks.shape, (L, R, Hkv, d))
    esz = k_cache.dtype.itemsize
    _load().oracle_kv_refresh(_p(k_cache), _p(v_cache), _p(k_src), _p(v_src), _p(pos),
                              ctypes.c_int(R), ctypes.c_int(kv_base_row), ctypes.c_int(L),
                              ctypes.c_int(Hkv), ctypes.c_int64(cache_rows), ctypes.c_int64(d * esz),
                              ctypes.c_int64(Hkv * cache_rows * d * esz),
                              ctypes.c_int64(R * Hkv * d * esz))


def confidence_select(logits, tokens_in, mask_id: int, eos_id: int, threshold: float,
                      lanes=None, force_top1: bool = False):
    """O-C.  logits [N,V]; returns dict(conf f64[N], argmax i32[N], p2 f64[N], commit u8[N],
    tokens_out i32[N])."""
    logits = _f32(logits)
    N, V = logits.shape
    tokens_in = _i32(tokens_in)
    assert tokens_in.shape == (N,)
    lanes_arr = None if lanes is None else _i32(lanes).reshape(-1, 6)
    conf = np.zeros(N, np.float64)
    p2 = np.zeros(N, np.float64)
    argmax = np.zeros(N, np.int32)
    commit = np.zeros(N, np.uint8)
    tokens_out = np.zeros(N, np.int32)
    _load().oracle_confidence_select(_p(logits), ctypes.c_int(N), ctypes.c_int(V), ctypes.c_int64(V),
                                     _p(tokens_in), ctypes.c_int(mask_id), ctypes.c_int(eos_id),
                                     ctypes.c_double(threshold), _p(lanes_arr),
                                     ctypes.c_int(0 if lanes_arr is None else lanes_arr.shape[0]),
                                     ctypes.c_int(1 if force_top1 else 0), _p(conf), _p(argmax),
                                     _p(p2), _p(commit), _p(tokens_out))
    return dict(conf=conf, argmax=argmax, p2=p2, commit=commit, tokens_out=tokens_out)


def lane_status(lanes, tokens_in, conf, argmax, mask_id: int, eos_id: int, tau_future: float,
                delimiters, no_fork_prev, commit, tokens_out):
    """O-D.  Per-lane integers after the transfer + the lookahead draft rule (Eq.8).  `commit` and
    `tokens_out` are the select's outputs; copies are returned with the lookahead rows decided by Eq.8.
    Returns dict(status int32 [n,8] = n_filled, valid_prefix, split_point, n_committed, n_drafts, n_masked, 0, 0;
    commit u8[N]; tokens_out i32[N])."""
    lanes = _i32(lanes).reshape(-1, 6)
    tokens_in = _i32(tokens_in)
    N = tokens_in.shape[0]
    conf = np.ascontiguousarray(conf, dtype=np.float64)
    argmax = _i32(argmax)
    delimiters, no_fork_prev = _i32(delimiters).reshape(-1), _i32(no_fork_prev).reshape(-1)
    commit_io = np.ascontiguousarray(commit, dtype=np.uint8).copy()
    tokens_io = _i32(tokens_out).copy()
    status = np.zeros((lanes.shape[0], 8), np.int32)
    _load().oracle_lane_status(_p(lanes), ctypes.c_int(lanes.shape[0]), ctypes.c_int(N), _p(tokens_in), _p(conf),
                               _p(argmax), ctypes.c_int(mask_id), ctypes.c_int(eos_id), ctypes.c_double(tau_future),
                               _p(delimiters) if delimiters.size else None, ctypes.c_int(delimiters.size),
                               _p(no_fork_prev) if no_fork_prev.size else None, ctypes.c_int(no_fork_prev.size),
                               _p(commit_io), _p(tokens_io), _p(status))
    return dict(status=status, commit=commit_io, tokens_out=tokens_io)


def refresh_forward(q, k_new, v_new, k_cache, v_cache, lanes, scale: Optional[float] = None):
    """O-E.  Attention of every lane over [its prefix ; its own rows] (O-A), then the lanes' K_new/V_new rows
    written into the caches behind their prefixes, IN PLACE on k_cache / v_cache (float32 [Hkv,cache_rows,d]).
    Returns (out fp64 [T,Hq,d], lse fp64 [T,Hq])."""
    q, k_new, v_new = map(_f32, (q, k_new, v_new))
    assert k_cache.dtype == np.float32 and v_cache.dtype == np.float32
    assert k_cache.flags["C_CONTIGUOUS"] and v_cache.flags["C_CONTIGUOUS"]
    lanes = _i32(lanes).reshape(-1, 6)
    T, Hq, d = q.shape
    Hkv, cache_rows = k_cache.shape[0], k_cache.shape[1]
    if scale is None:
        scale = 1.0 / np.sqrt(float(d))
    out = np.zeros((T, Hq, d), dtype=np.float64)
    lse = np.zeros((T, Hq), dtype=np.float64)
    _load().oracle_refresh_forward(_p(q), _p(k_new), _p(v_new), _p(k_cache), _p(v_cache), _p(lanes),
                                   ctypes.c_int(lanes.shape[0]), ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d),
                                   ctypes.c_int64(cache_rows), ctypes.c_double(scale), _p(out), _p(lse))
    return out, lse


def lm_head_confidence(hidden, weight, tokens_in, mask_id: int, eos_id: int, threshold: float, lanes=None,
                       force_top1: bool = False):
    """O-F.  hidden [N,K], weight [V,K] (float32 values already rounded to the I/O dtype); logits = hidden @ weight.T
    in fp64, consumed by the rule of O-C.  Returns the same dict as confidence_select."""
    hidden, weight = _f32(hidden), _f32(weight)
    N, K = hidden.shape
    V = weight.shape[0]
    assert weight.shape == (V, K)
    tokens_in = _i32(tokens_in)
    lanes_arr = None if lanes is None else _i32(lanes).reshape(-1, 6)
    conf, p2 = np.zeros(N, np.float64), np.zeros(N, np.float64)
    argmax, commit, tokens_out = np.zeros(N, np.int32), np.zeros(N, np.uint8), np.zeros(N, np.int32)
    _load().oracle_lm_head_confidence(_p(hidden), _p(weight), ctypes.c_int(N), ctypes.c_int(V), ctypes.c_int(K),
                                      _p(tokens_in), ctypes.c_int(mask_id), ctypes.c_int(eos_id),
                                      ctypes.c_double(threshold), _p(lanes_arr),
                                      ctypes.c_int(0 if lanes_arr is None else lanes_arr.shape[0]),
                                      ctypes.c_int(1 if force_top1 else 0), _p(conf), _p(argmax), _p(p2), _p(commit),
                                      _p(tokens_out))
    return dict(conf=conf, argmax=argmax, p2=p2, commit=commit, tokens_out=tokens_out)
