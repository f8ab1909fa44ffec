"""CPU-only pins of oracle.lane_status (O-D: SURVEY 8(f) NEXT-2 -- the lookahead draft rule Eq.8 PAPER.md
L108, fill ratio Eq.5, valid prefix Eq.9, split point Eq.4): a hand-worked example, closed
forms, a brute-force re-derivation in set/array form, and invariants chosen so that a wrong index base,
a dropped exclusion or a swapped comparison fails one of them."""
import json
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
MASK, EOS = 99, 2


def lanes_of(specs):
    """specs: (q_start, b, w, refine) -> int32 [n, 6] with the lookahead window in flags bits 8..23"""
    return np.array([[0, 0, 0, s, b + w, (w << 8) | (1 if r else 0)] for s, b, w, r in specs], np.int32)


def run(lanes, tokens_in, tokens_sel, commit_sel, conf, argmax, tau_future=0.9, delims=(7,), nofork=(5,)):
    return oracle.lane_status(lanes, tokens_in, conf, argmax, MASK, EOS, tau_future, list(delims), list(nofork),
                              commit_sel, tokens_sel)


def test_hand_worked_example():
    g = json.load(open(os.path.join(HERE, "golden", "lane_status_example.json")))
    r = oracle.lane_status(np.array(g["lanes"], np.int32), g["tokens_in"], g["conf"], g["argmax"], g["mask_id"],
                           g["eos_id"], g["tau_future"], g["delimiters"], g["no_fork_prev"],
                           g["commit_after_select"], g["tokens_after_select"])
    assert r["status"].tolist() == g["expected_status"]
    assert r["tokens_out"].tolist() == g["expected_tokens_out"]
    assert r["commit"].tolist() == g["expected_commit"]


def test_closed_forms_valid_prefix_and_fill():
    b = 12
    z = np.arange(20, 20 + b, dtype=np.int32)                       # no MASK, no EOS, no delimiter
    zero = np.zeros(b, np.uint8)
    r = run(lanes_of([(0, b, 0, False)]), z, z, zero, np.full(b, 0.5), z)
    assert r["status"][0].tolist() == [b, b, 0, 0, 0, 0, 0, 0]     # v = b (Eq.9: the {b} member), p = 0: no delimiter
    z2 = z.copy(); z2[0] = MASK
    assert run(lanes_of([(0, b, 0, False)]), z2, z2, zero, np.full(b, 0.5), z)["status"][0, 1] == 0   # first token MASK -> v = 0
    z3 = z.copy(); z3[5] = EOS; z3[3] = MASK
    st = run(lanes_of([(0, b, 0, False)]), z3, z3, zero, np.full(b, 0.5), z)["status"][0]
    assert st[1] == 3 and st[0] == b - 1 and st[5] == 1             # the EARLIER of MASK / EOS; EOS counts as filled
    z4 = z.copy(); z4[b - 1] = 7                                    # a delimiter in the last position: p = b
    assert run(lanes_of([(0, b, 0, False)]), z4, z4, zero, np.full(b, 0.5), z)["status"][0, 2] == b


def test_split_point_takes_the_last_valid_delimiter_and_applies_the_exclusion():
    z = np.array([7, 30, 7, 5, 7, 31, 5, 7], np.int32)              # delimiters at 0, 2, 4 (after a 5), 7 (after a 5)
    zero = np.zeros(8, np.uint8)
    lanes = lanes_of([(0, 8, 0, False)])
    assert run(lanes, z, z, zero, np.full(8, 0.5), z)["status"][0, 2] == 3          # 4 and 7 excluded -> i = 2
    assert run(lanes, z, z, zero, np.full(8, 0.5), z, nofork=())["status"][0, 2] == 8   # no exclusion -> i = 7
    assert run(lanes, z, z, zero, np.full(8, 0.5), z, delims=())["status"][0, 2] == 0   # empty delimiter set
    assert run(lanes, z, z, zero, np.full(8, 0.5), z, delims=(7, 31))["status"][0, 2] == 6   # 31 at i = 5 is valid


def test_lookahead_rule_threshold_mask_and_eos():
    """Eq.8: drafted iff MASK in, q >= tau_future (>=, checked at equality), greedy token not EOS."""
    lanes = lanes_of([(0, 2, 5, False)])
    tin = np.array([40, 41, MASK, MASK, MASK, 17, MASK], np.int32)
    conf = np.array([0.5, 0.5, 0.9, 0.8999, 0.99, 0.99, 0.95])
    am = np.array([40, 41, 50, 51, EOS, 52, 53], np.int32)
    sel_tok = tin.copy(); sel_tok[2:] = [60, 61, 62, 63, 64]         # whatever the transfer rule wrote is overridden
    sel_commit = np.array([0, 0, 1, 1, 1, 1, 1], np.uint8)
    r = run(lanes, tin, sel_tok, sel_commit, conf, am, tau_future=0.9)
    assert r["tokens_out"].tolist() == [40, 41, 50, MASK, MASK, 17, 53]
    assert r["commit"].tolist() == [0, 0, 1, 0, 0, 0, 1]
    assert r["status"][0, 4] == 2
    assert run(lanes, tin, sel_tok, sel_commit, conf, am, tau_future=1.5)["status"][0, 4] == 0
    assert run(lanes, tin, sel_tok, sel_commit, conf, am, tau_future=0.0)["status"][0, 4] == 3   # EOS still rejected


def brute_force(lanes, tokens_in, tokens_sel, commit_sel, conf, argmax, tau, delims, nofork):
    """The same quantities from set / array formulations (no per-lane running minimum or maximum)."""
    tok = np.array(tokens_sel, np.int32).copy(); com = np.array(commit_sel, np.uint8).copy()
    out = []
    for lane in lanes:
        s, n, w = int(lane[3]), int(lane[4]), (int(lane[5]) >> 8) & 0xffff
        b = n - w
        la = np.arange(s + b, s + n)
        c = (np.asarray(tokens_in)[la] == MASK) & (np.asarray(conf)[la] >= tau) & (np.asarray(argmax)[la] != EOS)
        tok[la] = np.where(c, np.asarray(argmax)[la], np.asarray(tokens_in)[la]); com[la] = c
        z = tok[s:s + b]
        stops = set(np.nonzero((z == MASK) | (z == EOS))[0].tolist()) | {b}
        prev_ok = np.concatenate([[True], ~np.isin(z[:-1], list(nofork))]) if b else np.zeros(0, bool)
        cand = [i + 1 for i in range(b) if z[i] in set(delims) and prev_ok[i]]
        out.append([int((z != MASK).sum()), min(stops), max(cand) if cand else 0, int(com[s:s + b].sum()), int(c.sum()),
                    int((z == MASK).sum()), 0, 0])
    return np.array(out, np.int32), tok, com


@pytest.mark.parametrize("seed", range(6))
def test_against_brute_force_on_random_lanes(seed):
    rng = np.random.default_rng(4000 + seed)
    specs, start = [], 0
    for _ in range(int(rng.integers(1, 9))):
        b, w = int(rng.integers(1, 40)), int(rng.integers(0, 9)) * int(rng.integers(0, 2))
        specs.append((start, b, w, bool(rng.integers(0, 2)))); start += b + w + int(rng.integers(0, 3))
    lanes = lanes_of(specs)
    N = start + 2
    vocab = [MASK, EOS, 5, 7, 8, 30, 31, 32]
    tin = rng.choice(vocab, size=N, p=[.4, .05, .1, .1, .05, .1, .1, .1]).astype(np.int32)
    conf = rng.random(N); am = rng.choice(vocab[1:], size=N).astype(np.int32)
    com = ((tin == MASK) & (conf >= 0.6)).astype(np.uint8); sel = np.where(com, am, tin).astype(np.int32)
    r = oracle.lane_status(lanes, tin, conf, am, MASK, EOS, 0.8, [7, 8], [5], com, sel)
    st, tok, c2 = brute_force(lanes, tin, sel, com, conf, am, 0.8, (7, 8), (5,))
    assert r["status"].tolist() == st.tolist()
    assert r["tokens_out"].tolist() == tok.tolist() and r["commit"].tolist() == c2.tolist()
    # invariants: n_filled + n_masked = b; v <= b; p <= b; rows outside the lanes untouched
    b = lanes[:, 4] - ((lanes[:, 5] >> 8) & 0xffff)
    assert (r["status"][:, 0] + r["status"][:, 5] == b).all()
    assert (r["status"][:, 1] <= b).all() and (r["status"][:, 2] <= b).all()
    covered = np.zeros(N, bool)
    for l in lanes:
        covered[l[3]:l[3] + l[4]] = True
    assert np.array_equal(r["tokens_out"][~covered], sel[~covered])


def test_drafts_are_monotone_in_tau_future():
    rng = np.random.default_rng(7)
    lanes = lanes_of([(0, 4, 28, False)])
    tin = np.full(32, MASK, np.int32); conf = rng.random(32); am = rng.integers(3, 50, 32).astype(np.int32)
    zero = np.zeros(32, np.uint8)
    counts = [int(run(lanes, tin, tin, zero, conf, am, tau_future=t)["status"][0, 4]) for t in (0.0, 0.3, 0.6, 0.9, 1.1)]
    assert counts == sorted(counts, reverse=True) and counts[0] == 28 and counts[-1] == 0
