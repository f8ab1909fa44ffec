"""CPU-only pins of oracle.refresh_forward (O-E: SURVEY 8(f) NEXT-3, Eq.12): the dense special
case against a library routine, the cache bytes against an array assignment, and the consistency that makes the
call what Eq.12 says it is -- after it, the cache HOLDS the states the range was attended with."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_08411_b200 import workloads as W


def rnd(rng, *shape):
    return rng.standard_normal(shape).astype(np.float32)


def test_prefix_zero_is_plain_bidirectional_self_attention_and_a_transposed_copy():
    rng = np.random.default_rng(1)
    Lr, Hq, Hkv, d, rows = 37, 4, 2, 16, 64
    q, k, v = rnd(rng, Lr, Hq, d), rnd(rng, Lr, Hkv, d), rnd(rng, Lr, Hkv, d)
    kc, vc = rnd(rng, Hkv, rows, d), rnd(rng, Hkv, rows, d)
    k0, v0 = kc.copy(), vc.copy()
    lanes = np.array([[0, 5, 0, 0, Lr, 0]], np.int32)                      # Eq.12: range [0, L_refresh) at base row 5
    out, lse = oracle.refresh_forward(q, k, v, kc, vc, lanes)
    tq = torch.from_numpy(q).double().permute(1, 0, 2)[None]
    tk = torch.from_numpy(k).double().permute(1, 0, 2)[None]
    tv = torch.from_numpy(v).double().permute(1, 0, 2)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=False, enable_gqa=True)[0].permute(1, 0, 2)
    assert np.abs(out - ref.numpy()).max() <= 1e-12
    assert np.array_equal(kc[:, 5:5 + Lr], k.transpose(1, 0, 2)) and np.array_equal(vc[:, 5:5 + Lr], v.transpose(1, 0, 2))
    untouched = np.ones(rows, bool); untouched[5:5 + Lr] = False
    assert np.array_equal(kc[:, untouched], k0[:, untouched]) and np.array_equal(vc[:, untouched], v0[:, untouched])


def test_the_cache_then_holds_the_states_the_range_was_attended_with():
    """A probe lane that sees the refreshed rows THROUGH THE CACHE gets what it would get seeing them as new rows."""
    rng = np.random.default_rng(2)
    Hq, Hkv, d, rows, pre, Lr = 4, 2, 8, 96, 11, 29
    kc, vc = rnd(rng, Hkv, rows, d), rnd(rng, Hkv, rows, d)
    q, k, v = rnd(rng, Lr + 3, Hq, d), rnd(rng, Lr + 3, Hkv, d), rnd(rng, Lr + 3, Hkv, d)
    lanes = np.array([[0, 2, pre, 0, Lr, 0]], np.int32)                    # an older prefix of 11 rows is kept
    kc2, vc2 = kc.copy(), vc.copy()
    out, _ = oracle.refresh_forward(q[:Lr], k[:Lr], v[:Lr], kc2, vc2, lanes)
    plain, _ = oracle.lane_attention(q[:Lr], k[:Lr], v[:Lr], kc, vc, lanes)
    assert np.array_equal(out, plain)                                      # the attention part IS O-A, on the old cache
    # probe: 3 new rows attending to [prefix of pre + Lr rows in the refreshed cache ; themselves]
    probe = np.array([[0, 2, pre + Lr, 0, 3, 0]], np.int32)
    via_cache, _ = oracle.lane_attention(q[Lr:], k[Lr:], v[Lr:], kc2, vc2, probe)
    # the same keys assembled by hand: old prefix, then the refreshed range, then the probe's own rows
    K = np.concatenate([kc[:, 2:2 + pre], k[:Lr].transpose(1, 0, 2), k[Lr:].transpose(1, 0, 2)], 1).astype(np.float64)
    Vv = np.concatenate([vc[:, 2:2 + pre], v[:Lr].transpose(1, 0, 2), v[Lr:].transpose(1, 0, 2)], 1).astype(np.float64)
    for h in range(Hq):
        s = q[Lr:, h].astype(np.float64) @ K[h // 2].T / np.sqrt(d)
        p = np.exp(s - s.max(-1, keepdims=True)); p /= p.sum(-1, keepdims=True)
        assert np.abs(via_cache[:, h] - p @ Vv[h // 2]).max() <= 1e-12


def test_several_ranges_in_one_call_and_idempotence():
    rng = np.random.default_rng(3)
    Hq, Hkv, d, rows = 2, 1, 8, 80
    lanes = np.array([[0, 0, 0, 0, 20, 0], [1, 40, 4, 20, 9, 0]], np.int32)
    q, k, v = rnd(rng, 29, Hq, d), rnd(rng, 29, Hkv, d), rnd(rng, 29, Hkv, d)
    kc, vc = rnd(rng, Hkv, rows, d), rnd(rng, Hkv, rows, d)
    o1, l1 = oracle.refresh_forward(q, k, v, kc, vc, lanes)
    snap = kc.copy()
    o2, l2 = oracle.refresh_forward(q, k, v, kc, vc, lanes)               # same states again: cache unchanged,
    assert np.array_equal(kc, snap)
    assert np.array_equal(o1[:20], o2[:20])                                # prefix-0 range: same output
    assert np.array_equal(kc[0, 44:53], k[20:, 0]) and np.array_equal(kc[0, :20], k[:20, 0])
