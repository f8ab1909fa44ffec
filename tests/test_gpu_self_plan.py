"""Self-planned attention launches (K1, "self-planned launches"): a small call -- at most 32 lanes, every
item a CTA of its own by the host's bounds, no item longer than 24 key tiles -- launches no plan kernel; every CTA
of the attention kernel derives its record from the lane descriptors.  The record is the one lane_plan_kernel's
whole-item branch writes, so the outputs must be BIT-identical to those of a handle that always runs the plan
kernel (ASYNCLANE_SELF_PLAN=0 at al_create), one launch less; parity with the oracle is test_gpu_parity's."""
import os

import pytest

torch = pytest.importorskip("torch")

import oracle
import numpy as np
from paper_2606_08411_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handles():
    from paper_2606_08411_b200 import binding
    h_self = binding.Handle(0)
    os.environ["ASYNCLANE_SELF_PLAN"] = "0"
    try:
        h_plan = binding.Handle(0)
    finally:
        del os.environ["ASYNCLANE_SELF_PLAN"]
    yield h_self, h_plan
    h_self.close(); h_plan.close()


def small(name, seed, Hq, Hkv, groups, cache_rows=1400):
    return W.build_workload(name, seed, "bf16", Hq, Hkv, 128, 1, cache_rows, groups, n_refresh=1, refresh_base_row=0,
                            refresh_span=8, vocab=64, logit_sigma=1.0, planted_frac=0.0, mask_id=63, eos_id=-1,
                            threshold=0.9)


CASES = {
    "cfg2": lambda: W.cfg2_llada_layer(),
    "cfg3": lambda: W.cfg3_dream_layer(),
    "ragged": lambda: W.ragged_case(101),
    "one lane, one row": lambda: small("one_row", 41, 4, 2, [dict(kv_base_row=3, prefix_len=70, q_lens=[1])]),
    "no prefix": lambda: small("no_prefix", 42, 4, 4, [dict(kv_base_row=0, prefix_len=0, q_lens=[32, 5])]),
    "per-lane prefixes, two runs, n_rep 7": lambda: small(
        "mixed", 43, 7, 1, [dict(kv_base_row=0, prefix_len=[257, 129, 1], q_lens=[32, 17, 32]),
                            dict(kv_base_row=300, prefix_len=128, q_lens=[24])]),
    "n_rep 16: eight tokens per sub-tile, 9 tiles in a run": lambda: small(
        "nrep16", 44, 16, 1, [dict(kv_base_row=0, prefix_len=300, q_lens=[32, 32, 7])]),
    "32 lanes in 8 runs (the most a warp plans)": lambda: small(
        "lanes32", 45, 2, 1, [dict(kv_base_row=130 * i, prefix_len=[100 + i, 90, 64, 3], q_lens=[3, 1, 2, 1])
                              for i in range(8)]),
    "two sub-tiles per tile (one each would take more CTAs than a quarter of the grid)": lambda: small(
        "two_sub", 46, 8, 8, [dict(kv_base_row=0, prefix_len=200, q_lens=[110] * 10)]),
}


@pytest.mark.parametrize("name", list(CASES))
def test_self_planned_equals_plan_kernel(handles, name):
    from paper_2606_08411_b200.step import LaneStep
    h_self, h_plan = handles
    wl = CASES[name]()
    outs, launches = [], []
    for h in (h_self, h_plan):
        st = LaneStep(h, wl)
        n0 = h.al_launch_count
        st.attention()
        torch.cuda.synchronize()
        launches.append(h.al_launch_count - n0)
        outs.append((st.out.clone(), st.lse.clone()))
    assert launches == [wl.n_layers, wl.n_layers + 1], launches       # the plan kernel is the launch that went away
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    ref, ref_lse = oracle.lane_attention(wl.q[0], wl.k_new[0], wl.v_new[0], wl.k_cache[0], wl.v_cache[0], wl.lanes)
    covered = np.zeros(wl.total_q_rows, bool)
    for l in wl.lanes:
        covered[l[W.LANE_Q_START]:l[W.LANE_Q_START] + l[W.LANE_Q_LEN]] = True
    out = outs[0][0][0].float().cpu().numpy()
    err = (np.abs(out - ref).max(-1) / np.maximum(np.abs(ref).max(-1), 1e-30))[covered].max()
    assert err <= 1e-2, err


def test_calls_outside_the_bounds_still_run_the_plan_kernel(handles):
    """More than 32 lanes, more possible items than CTAs, or a prefix bound beyond 24 key tiles: plan kernel."""
    from paper_2606_08411_b200.step import LaneStep
    h_self, _ = handles
    for wl in (small("lanes33", 47, 2, 1, [dict(kv_base_row=0, prefix_len=64, q_lens=[1] * 33)]),
               W.cfg4_long_llada(n_layers=1),
               small("long", 48, 2, 1, [dict(kv_base_row=0, prefix_len=2100, q_lens=[32])], cache_rows=2200)):
        st = LaneStep(h_self, wl)
        n0 = h_self.al_launch_count
        st.attention()
        torch.cuda.synchronize()
        assert h_self.al_launch_count - n0 == wl.n_layers + 1
