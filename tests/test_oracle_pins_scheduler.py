"""CPU-only pins of oracle.scheduler (Alg.1).  The paper prints no worked
trace, so the pins are what the algorithm fixes whatever the schedule: the decoded text (the stub model's greedy
token is the target at every position, so ANY correct schedule must reproduce the target up to EOS), the
block-wise special case (no delimiters, no lookahead: Alg.1 degenerates to synchronous block decoding, whose
iteration count has a closed form), tree invariants of the fork operator, and the NFE accounting of Eq.11/13."""
import numpy as np
import pytest

from oracle import scheduler as S
from paper_2606_08411_b200 import workloads as W


def blockwise(case):
    cfg = dict(case["cfg"]); cfg["delimiter_ids"] = []; cfg["lookahead"] = 0
    return cfg


def commit_step(case, pos):
    """first local step t (0-based) at which position `pos` reaches q >= tau under the stub model (fp64)"""
    b = case["base"][pos].astype(np.float64); tgt = case["target"][pos]
    for t in range(200):
        x = b.copy(); x[tgt] += case["gain"] * (t + 1)
        if np.exp(x[tgt] - np.log(np.exp(x).sum())) >= case["cfg"]["tau"]:
            return t
    raise AssertionError


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_any_schedule_decodes_the_target_up_to_eos(seed):
    case = W.scheduler_case(seed)
    for cfg in (case["cfg"], blockwise(case), dict(case["cfg"], rho_min=0.0, t_min=0), dict(case["cfg"], lookahead=0)):
        r = S.run(cfg, case["base"], case["target"], case["gain"], case["prompt"])
        assert r["output"].tolist() == case["target"][:case["eos_at"]].tolist()
        assert all(n["state"] != S.ACTIVE for n in r["tree"])


def test_blockwise_special_case_has_the_closed_form_iteration_count():
    """No delimiters, no lookahead: one lane at a time, block after block.  A block's tokens commit at their own
    commit step or earlier (the forced token), the block completes when its last token commits, and the EOS block
    is followed by one more lane that stops the cascade (v = 0)."""
    case = W.scheduler_case(4, gen_len=96, block_size=32)
    r = S.run(blockwise(case), case["base"], case["target"], case["gain"], case["prompt"])
    assert r["stats"]["forks"] == 0 and all(n["role"] == S.GEN for n in r["tree"])
    starts = [n["start"] for n in r["tree"]]
    assert starts[:3] == [0, 32, 64]                        # successors start at s + v = s + B while no EOS shows
    # every lane's step count is bounded by its slowest position's commit step + 1 and by the forced-token rule
    for n in r["tree"]:
        slow = max(commit_step(case, g) for g in range(n["start"], n["start"] + n["len"]))
        assert n["steps"] <= slow + 1
    eos_block = case["eos_at"] // 32
    assert r["tree"][eos_block]["valid_prefix"] == case["eos_at"] - 32 * eos_block
    assert r["stats"]["stopped_frontiers"] == 1             # cascading termination: exactly one frontier stops
    assert r["stats"]["model_calls"] == r["stats"]["iterations"] == sum(n["steps"] for n in r["tree"])


@pytest.mark.parametrize("seed", [5, 6, 7, 8])
def test_fork_tree_invariants_and_accounting(seed):
    case = W.scheduler_case(seed, gen_len=200)
    r = S.run(case["cfg"], case["base"], case["target"], case["gain"], case["prompt"])
    tree, st = r["tree"], r["stats"]
    assert st["forks"] >= 1
    for i, n in enumerate(tree):
        if n["state"] == S.FORKED:
            ref, gen = tree[n["ref_child"]], tree[n["gen_child"]]
            assert ref["role"] == S.REF and gen["role"] == S.GEN and ref["parent"] == gen["parent"] == i
            assert ref["start"] == n["start"] and gen["start"] == n["start"] + ref["len"]      # Eq.6: split in place
            assert 0 < ref["len"] < n["len"]
            assert case["target"][n["start"] + ref["len"] - 1] == 7                            # Eq.4: ends on a delimiter
            assert n["start"] + ref["len"] - 2 < 0 or case["target"][n["start"] + ref["len"] - 2] != 5   # ValidBoundary
        if n["successor"] >= 0:
            assert tree[n["successor"]]["start"] == n["start"] + n["valid_prefix"] and n["valid_prefix"] > 0
        assert n["role"] == S.GEN or (n["ref_child"] < 0 and n["successor"] < 0)               # refine lanes are leaves
    assert st["lane_forwards"] >= st["model_calls"] == st["iterations"]                       # Eq.11: |G_t| <= |A_t|
    assert st["lane_forwards"] == sum(n["steps"] for n in tree)
    assert st["forks"] == sum(n["state"] == S.FORKED for n in tree)
    assert st["tokens_committed"] + st["tokens_drafted"] >= case["eos_at"]
    # asynchronous advancement (Eq.7): the continuation starts before its refine sibling finishes
    for n in tree:
        if n["state"] == S.FORKED and tree[n["ref_child"]]["steps"] > 1:
            assert tree[n["gen_child"]]["steps"] >= 1
    # refresh (Eq.12): L_refresh is monotone and never beyond P + L
    assert r["refreshed"] == sorted(r["refreshed"]) and r["refreshed"][-1] <= case["cfg"]["prompt_len"] + 200


def test_budget_exhaustion_leaves_a_truncated_but_consistent_output():
    case = W.scheduler_case(9)
    r = S.run(dict(case["cfg"], max_iterations=7), case["base"], case["target"], case["gain"], case["prompt"])
    out = r["output"].tolist()
    # unfinished leaves are cut at their first MASK, so the collected text is the target with holes: a subsequence
    it = iter(case["target"].tolist())
    assert all(any(t == u for u in it) for t in out) and 0 < len(out) < case["eos_at"]
    assert r["stats"]["iterations"] == 7 and any(n["state"] == S.ACTIVE for n in r["tree"])
    decoded = r["x"][case["cfg"]["prompt_len"]:]
    known = decoded != case["cfg"]["mask_id"]
    assert np.array_equal(decoded[known], case["target"][known])     # every committed token is the greedy target
