"""Pins for the CPU oracle (CPU only; `-m "not gpu"`).

The paper prints no numeric value for any attention output, cache row or confidence
(SURVEY.md section 4), so the oracle is pinned by what the paper's definitions and the
mathematics fix: brute force in NumPy on tiny inputs, closed forms (tests/golden/closed_forms.json,
hand-derived), library special cases (torch CPU SDPA, scipy logsumexp, numpy fancy indexing),
and structural invariants (lane independence, permutation, GQA == repeated MHA, split-LSE merge).
Each pin is chosen so that a plausible mistake (dropped term, wrong index, transposed operand,
lane leak, wrong comparison) fails at least one of them.
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2606_08411_b200 import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))


# --------------------------------------------------------------------------------------------
# helpers: an independent NumPy brute force (dense matrices, per lane) -- PAPER.md L70, Eq.2-3
# --------------------------------------------------------------------------------------------
def brute_lane_attention(q, k_new, v_new, k_cache, v_cache, lanes, scale=None):
    q, k_new, v_new, k_cache, v_cache = (np.asarray(a, np.float64) for a in (q, k_new, v_new, k_cache, v_cache))
    T, Hq, d = q.shape
    Hkv = k_cache.shape[0]
    n_rep = Hq // Hkv
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    out = np.zeros((T, Hq, d))
    lse = np.zeros((T, Hq))
    for (gid, base, plen, qs, ql, fl) in np.asarray(lanes).reshape(-1, 6):
        for h in range(Hq):
            g = h // n_rep
            K = np.concatenate([k_cache[g, base:base + plen], k_new[qs:qs + ql, g]], axis=0)
            V = np.concatenate([v_cache[g, base:base + plen], v_new[qs:qs + ql, g]], axis=0)
            S = scale * (q[qs:qs + ql, h] @ K.T)
            m = S.max(axis=1, keepdims=True)
            P = np.exp(S - m)
            Z = P.sum(axis=1, keepdims=True)
            out[qs:qs + ql, h] = (P / Z) @ V
            lse[qs:qs + ql, h] = (m + np.log(Z))[:, 0]
    return out, lse


def small_case(seed=0, Hq=4, Hkv=2, d=16, dtype="f32", n_groups=2):
    return W.ragged_case(seed, dtype=dtype, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=d,
                         n_groups=n_groups, vocab=257, max_prefix=50)


def run_attn(w, lanes=None, **kw):
    return oracle.lane_attention(w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0],
                                 w.lanes if lanes is None else lanes, **kw)


# --------------------------------------------------------------------------------------------
# O-A lane attention
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_attention_matches_numpy_brute_force(seed):
    w = small_case(seed)
    o, l = run_attn(w)
    bo, bl = brute_lane_attention(w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0], w.lanes)
    assert np.abs(o - bo).max() <= 1e-12
    assert np.abs(l - bl).max() <= 1e-12


def test_attention_cfg1_matches_brute_force():
    w = W.cfg1_tiny()
    o, l = run_attn(w)
    bo, bl = brute_lane_attention(w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0], w.lanes)
    assert np.abs(o - bo).max() <= 1e-12 and np.abs(l - bl).max() <= 1e-12


def test_attention_single_lane_equals_torch_sdpa_gqa():
    """One lane, no fork == plain non-causal block attention over [prefix || block]
    (library special case; also pins the GQA head mapping, reading C3)."""
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(7)
    Hq, Hkv, d, P, b = 6, 2, 32, 37, 13
    q = rng.standard_normal((b, Hq, d)).astype(np.float32)
    kn = rng.standard_normal((b, Hkv, d)).astype(np.float32)
    vn = rng.standard_normal((b, Hkv, d)).astype(np.float32)
    kc = rng.standard_normal((Hkv, 64, d)).astype(np.float32)
    vc = rng.standard_normal((Hkv, 64, d)).astype(np.float32)
    base = 5
    lanes = np.array([[0, base, P, 0, b, 0]], np.int32)
    o, _ = oracle.lane_attention(q, kn, vn, kc, vc, lanes)
    tq = torch.from_numpy(q).double().permute(1, 0, 2)[None]                       # [1,Hq,b,d]
    tk = torch.cat([torch.from_numpy(kc[:, base:base + P]), torch.from_numpy(kn).permute(1, 0, 2)], 1).double()[None]
    tv = torch.cat([torch.from_numpy(vc[:, base:base + P]), torch.from_numpy(vn).permute(1, 0, 2)], 1).double()[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=False, enable_gqa=True)
    ref = ref[0].permute(1, 0, 2).numpy()
    assert np.abs(o - ref).max() <= 1e-12


def test_attention_lane_independence_and_batched_equals_serial():
    """PAPER.md L70 "updated independently"; L168-172 grouping changes cost, not results."""
    w = small_case(11, n_groups=3)
    o, l = run_attn(w)
    for i in range(w.n_lanes):
        oi, li = run_attn(w, lanes=w.lanes[i:i + 1])
        qs, ql = w.lanes[i, W.LANE_Q_START], w.lanes[i, W.LANE_Q_LEN]
        assert np.array_equal(oi[qs:qs + ql], o[qs:qs + ql])          # bit-identical in the oracle
        assert np.array_equal(li[qs:qs + ql], l[qs:qs + ql])
    # perturbing lane 0's Q/K/V leaves every other lane bit-identical
    if w.n_lanes > 1:
        qs, ql = w.lanes[0, W.LANE_Q_START], w.lanes[0, W.LANE_Q_LEN]
        q2, k2, v2 = w.q[0].copy(), w.k_new[0].copy(), w.v_new[0].copy()
        q2[qs:qs + ql] += 1.0; k2[qs:qs + ql] -= 2.0; v2[qs:qs + ql] *= 3.0
        o2, _ = oracle.lane_attention(q2, k2, v2, w.k_cache[0], w.v_cache[0], w.lanes)
        rest = np.ones(o.shape[0], bool); rest[qs:qs + ql] = False
        assert np.array_equal(o2[rest], o[rest])
        assert not np.array_equal(o2[~rest], o[~rest])


def test_attention_rows_sum_to_one():
    w = small_case(12)
    v1 = np.ones_like(w.v_new[0]); c1 = np.ones_like(w.v_cache[0])
    o, _ = oracle.lane_attention(w.q[0], w.k_new[0], v1, w.k_cache[0], c1, w.lanes)
    assert np.abs(o - 1.0).max() <= 1e-13


def test_attention_zero_query_closed_form_visible_key_set():
    """Q == 0 => O = mean of the visible V rows: 35.5 / 39.5 (golden); a lane leak gives 42.3."""
    Hq = Hkv = 2; d = 32
    lanes = W.make_lanes([dict(kv_base_row=0, prefix_len=64, q_lens=[8, 8])])
    q = np.zeros((16, Hq, d), np.float32)
    rng = np.random.default_rng(0)
    kn = rng.standard_normal((16, Hkv, d)).astype(np.float32)
    kc = rng.standard_normal((Hkv, 96, d)).astype(np.float32)
    vc = np.zeros((Hkv, 96, d), np.float32)
    vc[:, :, :] = np.arange(96, dtype=np.float32)[None, :, None]       # row r valued r (rows >= 64 invisible)
    vn = np.zeros((16, Hkv, d), np.float32)
    vn[:8] = np.arange(64, 72, dtype=np.float32)[:, None, None]
    vn[8:] = np.arange(100, 108, dtype=np.float32)[:, None, None]
    o, lse = oracle.lane_attention(q, kn, vn, kc, vc, lanes)
    assert np.abs(o[:8] - GOLD["attention_zero_query_lane_A"]["value"]).max() <= 1e-12
    assert np.abs(o[8:] - GOLD["attention_zero_query_lane_B"]["value"]).max() <= 1e-12
    assert np.abs(o - GOLD["attention_zero_query_leak"]["value"]).min() > 1.0
    assert np.abs(lse - np.log(72.0)).max() <= 1e-13                    # LSE = ln(#visible keys)


def test_attention_prefix_permutation_and_lane_row_permutation():
    w = small_case(13, n_groups=1)
    o, _ = run_attn(w)
    base, plen = int(w.lanes[0, W.LANE_KV_BASE_ROW]), int(w.lanes[:, W.LANE_PREFIX_LEN].min())
    perm = np.random.default_rng(1).permutation(plen)
    kc, vc = w.k_cache[0].copy(), w.v_cache[0].copy()
    kc[:, base:base + plen] = kc[:, base + perm]; vc[:, base:base + plen] = vc[:, base + perm]
    o2, _ = oracle.lane_attention(w.q[0], w.k_new[0], w.v_new[0], kc, vc, w.lanes)
    assert np.abs(o2 - o).max() <= 1e-12
    # permuting the rows of one lane (Q, K_new, V_new jointly) permutes its outputs
    qs, ql = int(w.lanes[0, W.LANE_Q_START]), int(w.lanes[0, W.LANE_Q_LEN])
    p = np.random.default_rng(2).permutation(ql)
    q2, k2, v2 = w.q[0].copy(), w.k_new[0].copy(), w.v_new[0].copy()
    q2[qs:qs + ql] = q2[qs + p]; k2[qs:qs + ql] = k2[qs + p]; v2[qs:qs + ql] = v2[qs + p]
    o3, _ = oracle.lane_attention(q2, k2, v2, w.k_cache[0], w.v_cache[0], w.lanes)
    assert np.abs(o3[qs:qs + ql] - o[qs + p]).max() <= 1e-12


def test_attention_gqa_equals_mha_with_repeated_kv_heads():
    w = small_case(14, Hq=6, Hkv=2)
    o, l = run_attn(w)
    rep = 3
    o2, l2 = oracle.lane_attention(w.q[0], np.repeat(w.k_new[0], rep, axis=1), np.repeat(w.v_new[0], rep, axis=1),
                                   np.repeat(w.k_cache[0], rep, axis=0), np.repeat(w.v_cache[0], rep, axis=0), w.lanes)
    assert np.array_equal(o, o2) and np.array_equal(l, l2)


def test_attention_split_kv_lse_merge_invariance():
    """Any split of the key range merged by LSE equals the unsplit result (pins LSE; this is the
    identity the CUDA split-KV combine relies on)."""
    rng = np.random.default_rng(21)
    Hq = Hkv = 2; d = 16; P = 40; b = 9
    q = rng.standard_normal((b, Hq, d)).astype(np.float32)
    kn = rng.standard_normal((b, Hkv, d)).astype(np.float32); vn = rng.standard_normal((b, Hkv, d)).astype(np.float32)
    kc = rng.standard_normal((Hkv, P, d)).astype(np.float32); vc = rng.standard_normal((Hkv, P, d)).astype(np.float32)
    o, l = oracle.lane_attention(q, kn, vn, kc, vc, np.array([[0, 0, P, 0, b, 0]], np.int32))
    cut = 17
    # part 1: prefix rows [0,cut) only -> emulate with a lane of prefix cut and "own" keys removed:
    # use the brute force pieces via the oracle on re-packed inputs (prefix-only parts have q_len keys too,
    # so build the parts with numpy directly from the definition of LSE merging).
    bo1, bl1 = _part(q, kc[:, :cut], vc[:, :cut])
    bo2, bl2 = _part(q, np.concatenate([kc[:, cut:], kn.transpose(1, 0, 2)], 1), np.concatenate([vc[:, cut:], vn.transpose(1, 0, 2)], 1))
    m = np.maximum(bl1, bl2)
    w1, w2 = np.exp(bl1 - m), np.exp(bl2 - m)
    merged = (bo1 * w1[..., None] + bo2 * w2[..., None]) / (w1 + w2)[..., None]
    assert np.abs(merged - o).max() <= 1e-12
    assert np.abs(m + np.log(w1 + w2) - l).max() <= 1e-12


def _part(q, K, V):
    q = q.astype(np.float64); K = K.astype(np.float64); V = V.astype(np.float64)
    S = np.einsum("ihc,hjc->ihj", q, K) / np.sqrt(q.shape[-1])
    m = S.max(-1, keepdims=True); P = np.exp(S - m); Z = P.sum(-1, keepdims=True)
    return np.einsum("ihj,hjc->ihc", P / Z, V), (m + np.log(Z))[..., 0]


def test_attention_degenerate_prefix0_and_qlen1():
    rng = np.random.default_rng(5)
    Hq = Hkv = 1; d = 8
    q = rng.standard_normal((5, Hq, d)).astype(np.float32)
    kn = rng.standard_normal((5, Hkv, d)).astype(np.float32); vn = rng.standard_normal((5, Hkv, d)).astype(np.float32)
    kc = rng.standard_normal((Hkv, 10, d)).astype(np.float32); vc = rng.standard_normal((Hkv, 10, d)).astype(np.float32)
    # prefix_len = 0: pure block self-attention
    o, _ = oracle.lane_attention(q, kn, vn, kc, vc, np.array([[0, 3, 0, 0, 5, 0]], np.int32))
    S = (q[:, 0].astype(np.float64) @ kn[:, 0].astype(np.float64).T) / np.sqrt(d)
    P = np.exp(S - S.max(1, keepdims=True)); P /= P.sum(1, keepdims=True)
    assert np.abs(o[:, 0] - P @ vn[:, 0].astype(np.float64)).max() <= 1e-13
    # q_len = 1 lanes: single-query decode attention; its own key is always visible
    lanes = np.array([[0, 0, 10, i, 1, 0] for i in range(5)], np.int32)
    o1, _ = oracle.lane_attention(q, kn, vn, kc, vc, lanes)
    for i in range(5):
        K = np.concatenate([kc[0], kn[i]], 0).astype(np.float64); V = np.concatenate([vc[0], vn[i]], 0).astype(np.float64)
        s = K @ q[i, 0].astype(np.float64) / np.sqrt(d); p = np.exp(s - s.max()); p /= p.sum()
        assert np.abs(o1[i, 0] - p @ V).max() <= 1e-13


def test_attention_scale_argument_and_invariance():
    w = small_case(15)
    o, _ = run_attn(w)
    d = w.head_dim
    o2, _ = oracle.lane_attention(2.0 * w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0], w.lanes,
                                  scale=0.5 / np.sqrt(d))
    assert np.abs(o - o2).max() <= 1e-12
    o3, _ = run_attn(w, scale=1.0)          # a different scale must change the result
    assert np.abs(o - o3).max() > 1e-3


def test_attention_one_row_entry_point_equals_full():
    w = small_case(16)
    o, l = run_attn(w)
    for li in range(w.n_lanes):
        lane = w.lanes[li]
        for r in (0, int(lane[W.LANE_Q_LEN]) - 1):
            for h in range(w.n_q_heads):
                oo, ll = oracle.lane_attention_one(w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0], lane, r, h)
                row = int(lane[W.LANE_Q_START]) + r
                assert np.array_equal(oo, o[row, h]) and ll == l[row, h]
