"""Algorithmic work of one lane-batched denoising step.

These are the numerators of every roofline fraction bench.py reports: what the METHOD must do,
not what a kernel happens to move.  Masked padding, block-diagonal waste and split-KV partials are
deliberately not counted.
"""
from __future__ import annotations

from typing import Dict

import numpy as np

from .workloads import (LANE_GROUP_ID, LANE_PREFIX_LEN, LANE_Q_LEN, LaneStepWorkload)


def esize(dtype: str) -> int:
    return 2 if dtype == "bf16" else 4


def attention_flops_per_layer(wl: LaneStepWorkload) -> float:
    """4 H_q d sum_l q_len_l (prefix_len_l + q_len_l): QK^T and PV at 2 FLOP per MAC."""
    ql = wl.lanes[:, LANE_Q_LEN].astype(np.float64)
    pl = wl.lanes[:, LANE_PREFIX_LEN].astype(np.float64)
    return float(4.0 * wl.n_q_heads * wl.head_dim * np.sum(ql * (pl + ql)))


def attention_bytes_per_layer(wl: LaneStepWorkload) -> float:
    """K and V prefix rows ONCE PER GROUP + Q, O, K_new, V_new once."""
    e = esize(wl.dtype)
    per_group = 0
    for g in np.unique(wl.lanes[:, LANE_GROUP_ID]):
        per_group += int(wl.lanes[wl.lanes[:, LANE_GROUP_ID] == g, LANE_PREFIX_LEN].max())
    kv = 2.0 * wl.n_kv_heads * wl.head_dim * e * per_group
    io = float(wl.total_q_rows) * wl.head_dim * e * (2 * wl.n_q_heads + 2 * wl.n_kv_heads)
    return kv + io


def refresh_bytes(wl: LaneStepWorkload) -> float:
    """2 planes x (read + write) x R x H_kv x row bytes x layers + the index list."""
    R = int(wl.refresh_pos.size)
    return 2.0 * 2.0 * R * wl.n_kv_heads * wl.head_dim * esize(wl.dtype) * wl.n_layers + 4.0 * R


def confidence_bytes(wl: LaneStepWorkload) -> float:
    """logits once + tokens_in (4) + conf (4) + argmax (4) + commit (1) + tokens_out (4) per row."""
    N, V = wl.logits.shape
    return float(N) * V * esize(wl.dtype) + 17.0 * N


def summary(wl: LaneStepWorkload) -> Dict[str, float]:
    return dict(attn_flops=attention_flops_per_layer(wl) * wl.n_layers,
                attn_bytes=attention_bytes_per_layer(wl) * wl.n_layers,
                refresh_bytes=refresh_bytes(wl), confidence_bytes=confidence_bytes(wl),
                query_tokens=float(wl.total_q_rows))
