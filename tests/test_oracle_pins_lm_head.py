"""CPU-only pins of oracle.lm_head_confidence (O-F: SURVEY 8(f) NEXT-1, the LM head fused with the transfer rule of
PAPER.md L78-80 / Eq.8): against O-C on exactly representable products, against numpy + scipy, the identity
weight closed form, and the operand orientation (weight is [V][K])."""
import numpy as np
import pytest
from scipy.special import logsumexp

import oracle


def test_equals_o_c_on_the_materialised_logits_when_products_are_exact():
    rng = np.random.default_rng(1)
    N, K, V = 9, 16, 40
    h = rng.integers(-3, 4, (N, K)).astype(np.float32)           # small integers: every dot product is exact in fp32
    w = rng.integers(-2, 3, (V, K)).astype(np.float32) / 4.0
    logits = (h @ w.T).astype(np.float32)
    tokens = np.where(rng.random(N) < 0.6, 39, 3).astype(np.int32)
    lanes = np.array([[0, 0, 0, 0, 5, 1], [0, 0, 0, 5, 4, 0]], np.int32)
    for force in (False, True):
        a = oracle.lm_head_confidence(h, w, tokens, 39, 2, 0.3, lanes, force)
        b = oracle.confidence_select(logits, tokens, 39, 2, 0.3, lanes, force)
        for k in ("conf", "p2"):
            assert np.abs(a[k] - b[k]).max() <= 1e-14
        for k in ("argmax", "commit", "tokens_out"):
            assert np.array_equal(a[k], b[k])


def test_against_numpy_matmul_and_scipy_logsumexp():
    rng = np.random.default_rng(2)
    N, K, V = 6, 24, 300
    h, w = rng.standard_normal((N, K)).astype(np.float32), rng.standard_normal((V, K)).astype(np.float32)
    r = oracle.lm_head_confidence(h, w, np.full(N, 7, np.int32), 7, -1, 0.5)
    x = h.astype(np.float64) @ w.astype(np.float64).T
    assert np.array_equal(r["argmax"], x.argmax(1))
    assert np.abs(r["conf"] - np.exp(x.max(1) - logsumexp(x, axis=1))).max() <= 1e-13


def test_identity_weight_closed_form_and_orientation():
    """weight = a * I (V = K): logits = a * hidden.  hidden = e_j  ->  argmax j, conf = e^a / (e^a + V - 1)."""
    V = 32
    h = np.zeros((3, V), np.float32); h[0, 5] = 1; h[1, 31] = 1; h[2, 0] = 1
    r = oracle.lm_head_confidence(h, (8.0 * np.eye(V)).astype(np.float32), np.full(3, 9, np.int32), 9, -1, 0.9)
    assert r["argmax"].tolist() == [5, 31, 0]
    assert np.abs(r["conf"] - np.exp(8.0) / (np.exp(8.0) + V - 1)).max() <= 1e-14
    # a non-symmetric weight distinguishes [V][K] from [K][V]: row v of `weight` is the output direction of token v
    w = np.zeros((4, 2), np.float32); w[3] = [0, 5]; w[1] = [5, 0]
    r = oracle.lm_head_confidence(np.array([[1, 0], [0, 1]], np.float32), w, np.zeros(2, np.int32), 9, -1, 0.9)
    assert r["argmax"].tolist() == [1, 3]


def test_eos_suppression_only_on_refine_lanes():
    h = np.eye(4, dtype=np.float32)[[2, 2]]
    w = (6.0 * np.eye(4)).astype(np.float32)
    lanes = np.array([[0, 0, 0, 0, 1, 1], [0, 0, 0, 1, 1, 0]], np.int32)
    r = oracle.lm_head_confidence(h, w, np.full(2, 9, np.int32), 9, 2, 0.5, lanes)
    assert r["argmax"].tolist() == [0, 2]                        # refine row: EOS (id 2) removed, first of the rest wins
    assert r["conf"][0] == pytest.approx(1 / 3, abs=1e-12)
