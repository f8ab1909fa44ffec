"""GPU parity of al_refresh_forward (Eq.12) against oracle.refresh_forward:
attention outputs within the attention tolerance (1e-2 normwise, reading C10), refreshed cache rows bit-exact."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2606_08411_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handle():
    from paper_2606_08411_b200 import binding
    h = binding.Handle(0)
    yield h
    h.close()


def run_case(handle, Hq, Hkv, d, cache_rows, ranges, seed, dtype="bf16"):
    """ranges: (kv_base_row, prefix_len, q_len) per range, packed densely in q_start."""
    from paper_2606_08411_b200 import binding as B
    from paper_2606_08411_b200.step import to_device
    rng = np.random.default_rng(seed)
    rows, q_start = [], 0
    for gi, (base, pre, n) in enumerate(ranges):
        rows.append([gi, base, pre, q_start, n, 0]); q_start += n
    lanes = np.array(rows, np.int32)
    T = q_start
    rd = (lambda *s: W.round_to_bf16(rng.standard_normal(s).astype(np.float32))) if dtype == "bf16" else \
         (lambda *s: rng.standard_normal(s).astype(np.float32))
    q, k, v = rd(T, Hq, d), rd(T, Hkv, d), rd(T, Hkv, d)
    kc, vc = rd(Hkv, cache_rows, d), rd(Hkv, cache_rows, d)
    dev = torch.device("cuda:0")
    code = B.AL_BF16 if dtype == "bf16" else B.AL_F32
    shape = B.Handle.make_shape(Hq, Hkv, d, code, cache_rows)
    tq, tk, tv = to_device(q, dtype, dev), to_device(k, dtype, dev), to_device(v, dtype, dev)
    tkc, tvc = to_device(kc, dtype, dev), to_device(vc, dtype, dev)
    out = torch.zeros_like(tq); lse = torch.zeros(T, Hq, device=dev)
    maxp = int(lanes[:, 2].max())
    ws = torch.empty(max(16, handle.al_lane_attention_workspace_bytes(shape, len(lanes), T, maxp)), dtype=torch.uint8, device=dev)
    lanes_d = torch.from_numpy(lanes).to(dev)
    handle.al_refresh_forward(shape, tq, tk, tv, tkc, tvc, lanes_d, len(lanes), T, maxp, out, lse, ws)
    torch.cuda.synchronize()
    ref, ref_lse = oracle.refresh_forward(q, k, v, kc, vc, lanes)           # kc, vc refreshed in place
    o = out.float().cpu().numpy()
    err = (np.abs(o - ref).max(-1) / np.abs(ref).max(-1)).max()
    tol = 1e-2 if dtype == "bf16" else 2e-5
    assert err <= tol, err
    assert np.abs(lse.cpu().numpy() - ref_lse).max() <= (1e-3 if dtype == "bf16" else 2e-5)
    assert np.array_equal(tkc.float().cpu().numpy(), kc) and np.array_equal(tvc.float().cpu().numpy(), vc)


def test_eq12_dense_range_llada_shaped(handle):
    """prefix_len = 0, one range of L_refresh = 700 rows (not a multiple of any tile), 8 q / 2 kv heads"""
    run_case(handle, 8, 2, 128, 800, [(3, 0, 700)], seed=1)


def test_eq12_dream_shaped_gqa_and_mha(handle):
    run_case(handle, 28, 4, 128, 1100, [(0, 0, 1024)], seed=2)
    run_case(handle, 4, 4, 128, 600, [(0, 0, 513)], seed=3)


def test_batch_of_ranges_and_finalize_append(handle):
    """three sequences refreshed in one call, one of them keeping an older prefix (the Alg.1 line 16 append)"""
    run_case(handle, 8, 2, 128, 1500, [(0, 0, 300), (400, 0, 77), (600, 260, 45), (1000, 31, 1)], seed=4)


def test_fp32_path(handle):
    run_case(handle, 2, 2, 32, 200, [(5, 0, 60), (100, 20, 9)], seed=5, dtype="f32")
