"""GPU parity of al_lane_status (Eq.8 lookahead drafts, Eq.5 fill count, Eq.9 valid prefix,
Eq.4 split point) against oracle.lane_status -- integer work: bit-exact."""
import json
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2606_08411_b200 import workloads as W

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def handle():
    from paper_2606_08411_b200 import binding
    h = binding.Handle(0)
    yield h
    h.close()


def dev_i32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).cuda()


def run_status(handle, lanes, tokens_in, conf, argmax, mask_id, eos_id, tau, delims, nofork, commit_sel, tokens_sel):
    n_rows = len(tokens_in)
    lanes_d = dev_i32(lanes)
    commit = torch.from_numpy(np.ascontiguousarray(commit_sel, dtype=np.uint8)).cuda()
    tokens = dev_i32(tokens_sel)
    status = torch.full((len(lanes), 8), -7, dtype=torch.int32, device="cuda")
    handle.al_lane_status(lanes_d, len(lanes), n_rows, dev_i32(tokens_in),
                          torch.from_numpy(np.ascontiguousarray(conf, dtype=np.float32)).cuda(), dev_i32(argmax),
                          mask_id, eos_id, tau, dev_i32(delims) if len(delims) else None,
                          dev_i32(nofork) if len(nofork) else None, commit, tokens, status)
    torch.cuda.synchronize()
    return status.cpu().numpy(), commit.cpu().numpy(), tokens.cpu().numpy()


def test_hand_worked_example_on_gpu(handle):
    g = json.load(open(os.path.join(HERE, "golden", "lane_status_example.json")))
    st, com, tok = run_status(handle, np.array(g["lanes"], np.int32), g["tokens_in"], g["conf"], g["argmax"], g["mask_id"],
                              g["eos_id"], g["tau_future"], g["delimiters"], g["no_fork_prev"], g["commit_after_select"],
                              g["tokens_after_select"])
    assert st.tolist() == g["expected_status"]
    assert tok.tolist() == g["expected_tokens_out"] and com.tolist() == g["expected_commit"]


@pytest.mark.parametrize("seed", range(5))
def test_status_after_a_real_select_matches_the_oracle(handle, seed):
    """al_confidence_select, then al_lane_status on its outputs, against the oracle's two functions chained: lanes
    of 1..150 rows (several 32-row chunks), lookahead windows of 0..40 rows, refine lanes, delimiters on chunk edges."""
    rng = np.random.default_rng(5000 + seed)
    V, mask_id, eos_id = 96, 95, 2
    delims, nofork = [7, 8], [5, 6]
    rows, start = [], 0
    for g in range(int(rng.integers(2, 9))):
        b = int(rng.integers(1, 151)); refine = bool(rng.integers(0, 2))
        w = 0 if refine else int(rng.integers(0, 41)) * int(rng.integers(0, 2))
        rows.append([g, 0, 0, start, b + w, (w << 8) | int(refine)]); start += b + w
    lanes = np.array(rows, np.int32)
    N = start
    # logits whose greedy token is clearly decided and whose confidence is far from both thresholds
    x = (rng.standard_normal((N, V)) * 0.5).astype(np.float32)
    hot = rng.choice([2, 5, 6, 7, 8, 20, 21, 22, 23], size=N)
    peak = np.where(rng.random(N) < 0.6, 12.0, 3.0).astype(np.float32)
    x[np.arange(N), hot] += peak
    tokens = np.where(rng.random(N) < 0.6, mask_id, rng.choice([2, 5, 7, 8, 30, 31], size=N)).astype(np.int32)
    dev = torch.device("cuda:0")
    lg = torch.from_numpy(x).to(dev)
    conf = torch.zeros(N, device=dev); am = torch.zeros(N, dtype=torch.int32, device=dev)
    cm = torch.zeros(N, dtype=torch.uint8, device=dev); to = torch.zeros(N, dtype=torch.int32, device=dev)
    tin = dev_i32(tokens); lanes_d = dev_i32(lanes)
    handle.al_confidence_select(lg, N, V, V, tin, mask_id, eos_id, 0.9, lanes_d, len(lanes), 0, conf, am, cm, to, None)
    status = torch.zeros((len(lanes), 8), dtype=torch.int32, device=dev)
    handle.al_lane_status(lanes_d, len(lanes), N, tin, conf, am, mask_id, eos_id, 0.8, dev_i32(delims), dev_i32(nofork),
                          cm, to, status)
    torch.cuda.synchronize()
    r1 = oracle.confidence_select(x, tokens, mask_id, eos_id, 0.9, lanes)
    assert np.abs(r1["conf"] - 0.9).min() > 4e-3 and np.abs(r1["conf"] - 0.8).min() > 4e-3   # no row near a threshold
    r2 = oracle.lane_status(lanes, tokens, r1["conf"], r1["argmax"], mask_id, eos_id, 0.8, delims, nofork,
                            r1["commit"], r1["tokens_out"])
    assert np.array_equal(status.cpu().numpy(), r2["status"])
    assert np.array_equal(to.cpu().numpy(), r2["tokens_out"]) and np.array_equal(cm.cpu().numpy(), r2["commit"])
    assert int(r2["status"][:, 4].sum()) > 0 or not ((lanes[:, 5] >> 8) > 0).any()


def test_status_edge_cases_and_errors(handle):
    from paper_2606_08411_b200 import binding as B
    # a lane that is ALL lookahead (b = 0), a one-row lane, a 64-row lane with its only stop at row 63
    lanes = np.array([[0, 0, 0, 0, 5, 5 << 8], [0, 0, 0, 5, 1, 0], [1, 0, 0, 6, 64, 0]], np.int32)
    N = 70
    tin = np.full(N, 9, np.int32); tin[:5] = 1; tin[69] = 1
    conf = np.full(N, 0.99, np.float32); am = np.full(N, 4, np.int32)
    sel = tin.copy(); com = np.zeros(N, np.uint8)
    st, c2, tok = run_status(handle, lanes, tin, conf, am, 1, 2, 0.9, [9], [], com, sel)
    ref = oracle.lane_status(lanes, tin, conf, am, 1, 2, 0.9, [9], [], com, sel)
    assert np.array_equal(st, ref["status"]) and np.array_equal(tok, ref["tokens_out"]) and np.array_equal(c2, ref["commit"])
    assert st[0].tolist() == [0, 0, 0, 0, 5, 0, 0, 0] and st[1].tolist() == [1, 1, 1, 0, 0, 0, 0, 0]
    assert st[2, 1] == 63 and st[2, 2] == 63
    t = dev_i32(tin)
    with pytest.raises(B.AlError) as e:                      # tokens_io aliasing tokens_in is refused
        handle.al_lane_status(dev_i32(lanes), 3, N, t, torch.zeros(N, device="cuda"), dev_i32(am), 1, 2, 0.9, None, None,
                              torch.zeros(N, dtype=torch.uint8, device="cuda"), t,
                              torch.zeros((3, 8), dtype=torch.int32, device="cuda"))
    assert e.value.status == B.AL_ERR_INVALID_ARG
    handle.al_lane_status(dev_i32(lanes), 0, N, t, torch.zeros(N, device="cuda"), dev_i32(am), 1, 2, 0.9, None, None,
                          torch.zeros(N, dtype=torch.uint8, device="cuda"), dev_i32(sel),
                          torch.zeros((3, 8), dtype=torch.int32, device="cuda"))     # no lanes: valid no-op
