"""Pins for the CPU oracle, part 2: O-B compact refresh (Eq.12) and O-C
confidence / argmax / threshold select (Eq.8).  CPU only."""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2606_08411_b200 import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))


# --------------------------------------------------------------------------------------------
# O-B refresh
# --------------------------------------------------------------------------------------------
def _refresh_case(seed=0, L=3, Hkv=2, rows=40, d=8, R=7, dtype=np.float32, base=3):
    rng = np.random.default_rng(seed)
    kc = rng.standard_normal((L, Hkv, rows, d)).astype(dtype)
    vc = rng.standard_normal((L, Hkv, rows, d)).astype(dtype)
    pos = np.sort(rng.choice(rows - base, size=R, replace=False)).astype(np.int32)
    ks = rng.standard_normal((L, R, Hkv, d)).astype(dtype)
    vs = rng.standard_normal((L, R, Hkv, d)).astype(dtype)
    return kc, vc, ks, vs, pos, base


@pytest.mark.parametrize("dtype", [np.float32, np.uint16, np.float64])
def test_refresh_equals_numpy_fancy_index_assignment(dtype):
    kc, vc, ks, vs, pos, base = _refresh_case(1)
    kc, vc, ks, vs = (a.astype(dtype) if dtype != np.uint16 else (a * 100).astype(np.int64).astype(np.uint16)
                      for a in (kc, vc, ks, vs))
    ek, ev = kc.copy(), vc.copy()
    ek[:, :, base + pos, :] = ks.transpose(0, 2, 1, 3)
    ev[:, :, base + pos, :] = vs.transpose(0, 2, 1, 3)
    oracle.kv_refresh(kc, vc, ks, vs, pos, base)
    assert np.array_equal(kc.view(np.uint8), ek.view(np.uint8))
    assert np.array_equal(vc.view(np.uint8), ev.view(np.uint8))


def test_refresh_equals_torch_index_copy():
    torch = pytest.importorskip("torch")
    kc, vc, ks, vs, pos, base = _refresh_case(2)
    tk = torch.from_numpy(kc.copy()); tv = torch.from_numpy(vc.copy())
    idx = torch.from_numpy((base + pos).astype(np.int64))
    tk.index_copy_(2, idx, torch.from_numpy(ks).permute(0, 2, 1, 3).contiguous())
    tv.index_copy_(2, idx, torch.from_numpy(vs).permute(0, 2, 1, 3).contiguous())
    oracle.kv_refresh(kc, vc, ks, vs, pos, base)
    assert np.array_equal(kc, tk.numpy()) and np.array_equal(vc, tv.numpy())


def test_refresh_zero_positions_is_identity_and_idempotent():
    kc, vc, ks, vs, pos, base = _refresh_case(3)
    k0, v0 = kc.copy(), vc.copy()
    oracle.kv_refresh(kc, vc, ks[:, :0].copy(), vs[:, :0].copy(), pos[:0], base)
    assert np.array_equal(kc, k0) and np.array_equal(vc, v0)
    oracle.kv_refresh(kc, vc, ks, vs, pos, base)
    k1, v1 = kc.copy(), vc.copy()
    oracle.kv_refresh(kc, vc, ks, vs, pos, base)                  # idempotent
    assert np.array_equal(kc, k1) and np.array_equal(vc, v1)
    # untouched rows keep their bytes
    untouched = np.ones(kc.shape[2], bool); untouched[base + pos] = False
    assert np.array_equal(k1[:, :, untouched], k0[:, :, untouched])
    assert np.array_equal(v1[:, :, untouched], v0[:, :, untouched])
    assert not np.array_equal(k1[:, :, ~untouched], k0[:, :, ~untouched])


def test_refresh_all_rows_is_memcpy_and_joint_permutation_invariant():
    kc, vc, ks, vs, pos, base = _refresh_case(4, rows=12, R=12, base=0)
    assert np.array_equal(pos, np.arange(12))
    oracle.kv_refresh(kc, vc, ks, vs, pos, 0)
    assert np.array_equal(kc, ks.transpose(0, 2, 1, 3)) and np.array_equal(vc, vs.transpose(0, 2, 1, 3))
    # joint permutation of (pos, src) gives the same cache (positions unique)
    kc2, vc2, ks2, vs2, pos2, base2 = _refresh_case(5)
    a_k, a_v = kc2.copy(), vc2.copy()
    oracle.kv_refresh(a_k, a_v, ks2, vs2, pos2, base2)
    p = np.random.default_rng(0).permutation(pos2.size)
    b_k, b_v = kc2.copy(), vc2.copy()
    oracle.kv_refresh(b_k, b_v, np.ascontiguousarray(ks2[:, p]), np.ascontiguousarray(vs2[:, p]), pos2[p], base2)
    assert np.array_equal(a_k, b_k) and np.array_equal(a_v, b_v)


def test_refresh_composition_with_attention():
    """Refreshing rows >= every lane's prefix_len leaves attention unchanged; refreshing a visible
    row with new values changes it; refreshing a row with its current value is a no-op."""
    w = W.cfg1_tiny()
    o, _ = oracle.lane_attention(w.q[0], w.k_new[0], w.v_new[0], w.k_cache[0], w.v_cache[0], w.lanes)
    kc, vc = w.k_cache.copy(), w.v_cache.copy()
    pos = np.arange(64, 70, dtype=np.int32)                       # invisible rows (prefix_len = 64)
    rng = np.random.default_rng(9)
    ks = rng.standard_normal((1, 6, 2, 32)).astype(np.float32); vs = rng.standard_normal((1, 6, 2, 32)).astype(np.float32)
    oracle.kv_refresh(kc, vc, ks, vs, pos, 0)
    o2, _ = oracle.lane_attention(w.q[0], w.k_new[0], w.v_new[0], kc[0], vc[0], w.lanes)
    assert np.array_equal(o, o2)
    kc, vc = w.k_cache.copy(), w.v_cache.copy()
    oracle.kv_refresh(kc, vc, w.k_src, w.v_src, w.refresh_pos, w.refresh_base_row)     # visible rows
    o3, _ = oracle.lane_attention(w.q[0], w.k_new[0], w.v_new[0], kc[0], vc[0], w.lanes)
    assert np.abs(o3 - o).max() > 1e-6
    same_k = np.ascontiguousarray(kc[:, :, w.refresh_pos].transpose(0, 2, 1, 3))
    same_v = np.ascontiguousarray(vc[:, :, w.refresh_pos].transpose(0, 2, 1, 3))
    k4, v4 = kc.copy(), vc.copy()
    oracle.kv_refresh(k4, v4, same_k, same_v, w.refresh_pos, 0)
    assert np.array_equal(k4, kc) and np.array_equal(v4, vc)


# --------------------------------------------------------------------------------------------
# O-C confidence / select
# --------------------------------------------------------------------------------------------
def _conf(logits, tokens=None, mask_id=-7, eos_id=-1, tau=0.9, lanes=None, force=False):
    logits = np.asarray(logits, np.float32)
    if tokens is None:
        tokens = np.full(logits.shape[0], mask_id, np.int32)
    return oracle.confidence_select(logits, tokens, mask_id, eos_id, tau, lanes, force)


def test_confidence_closed_forms():
    V = 512
    r = _conf(np.full((1, V), 1.25))
    assert r["conf"][0] == pytest.approx(GOLD["confidence_all_equal_V512"]["value"], abs=1e-15)
    assert r["argmax"][0] == 0                                     # first maximiser (reading C6)
    row = np.zeros((1, V)); row[0, 137] = 8.0
    r = _conf(row)
    assert r["conf"][0] == pytest.approx(GOLD["confidence_single_peak_a8_V512"]["value"], abs=5e-7)   # golden has 6 digits
    assert r["conf"][0] == pytest.approx(np.exp(8.0) / (np.exp(8.0) + 511), abs=1e-13)
    assert r["argmax"][0] == 137 and r["commit"][0] == 0           # 0.8537 < 0.9
    a = GOLD["confidence_exact_0p9_logit_V512"]["value"]
    assert a == pytest.approx(np.log(9 * 511), abs=1e-7)
    row[0, 137] = a + 1e-3
    assert _conf(row)["commit"][0] == 1
    row[0, 137] = a - 1e-3
    assert _conf(row)["commit"][0] == 0


def test_confidence_threshold_comparison_is_ge():
    row = np.full((1, 64), -np.inf, np.float32); row[0, 3] = 0.0; row[0, 9] = 0.0
    r = _conf(row, tau=0.5)
    assert r["conf"][0] == GOLD["confidence_two_way_tie"]["value"]   # exactly 0.5
    assert r["commit"][0] == 1 and r["argmax"][0] == 3               # >= commits; lowest index wins the tie
    assert r["p2"][0] == 0.5
    assert _conf(row, tau=np.nextafter(0.5, 1.0))["commit"][0] == 0


def test_confidence_matches_scipy_logsumexp_and_probabilities_sum_to_one():
    sp = pytest.importorskip("scipy.special")
    w = W.cfg1_tiny()
    r = oracle.confidence_select(w.logits, w.tokens, w.mask_id, -1, w.threshold)
    x = w.logits.astype(np.float64)
    assert np.abs(r["conf"] - np.exp(x.max(1) - sp.logsumexp(x, axis=1))).max() <= 1e-14
    assert np.array_equal(r["argmax"], x.argmax(1))
    p = sp.softmax(x, axis=1)
    assert np.abs(p.sum(1) - 1).max() <= 1e-12
    assert np.abs(np.sort(p, 1)[:, -2] - r["p2"]).max() <= 1e-14
    # planted rows (and only they) exceed 0.9 (generator reading C9)
    assert set(np.nonzero(r["conf"] > 0.9)[0]) == set(w.planted_rows.tolist())


def test_confidence_shift_and_permutation_and_overflow():
    rng = np.random.default_rng(3)
    x = (rng.standard_normal((6, 300)) * 3).astype(np.float32).astype(np.float64)
    r = _conf(x)
    r2 = _conf(x + 2.0)                # +2.0 is exact in fp32 for these magnitudes? not guaranteed -> tolerance
    assert np.abs(r["conf"] - r2["conf"]).max() <= 1e-5 and np.array_equal(r["argmax"], r2["argmax"])
    perm = rng.permutation(300)
    r3 = _conf(x[:, perm])
    assert np.array_equal(perm[r3["argmax"]], r["argmax"])
    assert np.abs(r3["conf"] - r["conf"]).max() <= 1e-13
    big = x.copy(); big[:, 5] = 80.0 + x.max()
    r4 = _conf(big)
    assert np.all(np.isfinite(r4["conf"])) and np.all(r4["argmax"] == 5) and np.all(r4["conf"] > 0.999999)


def test_select_rules_masked_only_monotone_tau_and_token_write():
    w = W.cfg1_tiny()
    base = oracle.confidence_select(w.logits, w.tokens, w.mask_id, -1, 0.9)
    masked = w.tokens == w.mask_id
    assert np.array_equal(base["commit"].astype(bool), masked & (base["conf"] >= 0.9))
    assert np.array_equal(base["tokens_out"][~base["commit"].astype(bool)], w.tokens[~base["commit"].astype(bool)])
    assert np.array_equal(base["tokens_out"][base["commit"].astype(bool)], base["argmax"][base["commit"].astype(bool)])
    prev = None
    for tau in (1.5, 0.999, 0.9, 0.5, 0.1, 0.0, -1.0):
        c = oracle.confidence_select(w.logits, w.tokens, w.mask_id, -1, tau)["commit"].astype(bool)
        assert not np.any(c & ~masked)                              # unmasked rows never change
        if prev is not None:
            assert np.all(c | ~prev)                                # commit set grows as tau falls
        prev = c
    assert not oracle.confidence_select(w.logits, w.tokens, w.mask_id, -1, 1.5)["commit"].any()
    assert np.array_equal(oracle.confidence_select(w.logits, w.tokens, w.mask_id, -1, 0.0)["commit"].astype(bool), masked)


def test_select_eos_suppression_on_refine_lanes_only():
    """refine lanes suppress EOS; generate lanes allow it (reading C5)."""
    V = 32; eos = 4
    x = np.zeros((4, V), np.float32); x[:, eos] = 10.0; x[:, 7] = 9.0
    lanes = np.array([[0, 0, 0, 0, 2, W.LANE_FLAG_REFINE], [0, 0, 0, 2, 2, 0]], np.int32)
    r = _conf(x, eos_id=eos, lanes=lanes, tau=0.5)
    assert list(r["argmax"]) == [7, 7, eos, eos]
    # refine rows renormalise without the EOS entry
    z_ref = np.exp(9.0) + (V - 2)
    assert r["conf"][0] == pytest.approx(np.exp(9.0) / z_ref, abs=1e-14)
    z_gen = np.exp(10.0) + np.exp(9.0) + (V - 2)
    assert r["conf"][2] == pytest.approx(np.exp(10.0) / z_gen, abs=1e-14)
    # eos_id = -1 disables suppression
    r2 = _conf(x, eos_id=-1, lanes=lanes, tau=0.5)
    assert list(r2["argmax"]) == [eos] * 4


def test_select_force_top1_per_lane():
    V = 16
    x = np.zeros((6, V), np.float32)
    x[0, 1] = 1.0; x[1, 2] = 2.0; x[2, 3] = 2.0          # lane 0: nobody reaches tau; rows 1,2 tie on conf
    x[3, 4] = 9.0; x[4, 5] = 1.0; x[5, 6] = 0.5          # lane 1: row 3 commits by itself
    lanes = np.array([[0, 0, 0, 0, 3, 0], [0, 0, 0, 3, 3, 0]], np.int32)
    mask_id = 15
    tok = np.full(6, mask_id, np.int32)
    r = oracle.confidence_select(x, tok, mask_id, -1, 0.9, lanes, force_top1=True)
    assert list(r["commit"]) == [0, 1, 0, 1, 0, 0]        # lowest row wins the confidence tie
    assert list(r["tokens_out"]) == [mask_id, 2, mask_id, 4, mask_id, mask_id]
    r0 = oracle.confidence_select(x, tok, mask_id, -1, 0.9, lanes, force_top1=False)
    assert list(r0["commit"]) == [0, 0, 0, 1, 0, 0]
    # a lane whose best row is unmasked forces its best MASKED row; a lane with no masked row forces nothing
    tok2 = tok.copy(); tok2[1] = 3; tok2[3:] = 1
    r2 = oracle.confidence_select(x, tok2, mask_id, -1, 0.9, lanes, force_top1=True)
    assert list(r2["commit"]) == [0, 0, 1, 0, 0, 0]


def test_paper_accounting_consistency():
    g = GOLD["paper_accounting"]
    assert round(g["nfe"] / g["total_tokens"], 3) == g["nfe_per_token"]
