"""GPU parity of al_scheduler_run (Algorithm 1) against oracle.scheduler on
the same seeded stub-model inputs: the final token state, the collected output, every node of the lane tree and the
accounting must be identical (integer work).  The seeds are those whose oracle run keeps every decided confidence
more than 1e-4 away from both thresholds (fp32 on the GPU, fp64 in the oracle); the test checks that margin."""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import scheduler as S
from paper_2606_08411_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handle():
    from paper_2606_08411_b200 import binding
    h = binding.Handle(0)
    yield h
    h.close()


def compare(r, g):
    assert np.array_equal(g["x"], r["x"])
    assert g["output"].tolist() == r["output"].tolist()
    assert len(g["tree"]) == len(r["tree"])
    for a, b in zip(g["tree"], r["tree"]):
        assert a == {k: b[k] for k in a}, (a, b)
    assert g["stats"] == {k: r["stats"][k] for k in g["stats"]}


@pytest.mark.parametrize("seed,kw", [(21, {}), (23, {}), (24, {}), (28, {}), (35, {}), (37, {}),
                                      (21, dict(lookahead=0)), (23, dict(delimiter_ids=[])), (24, dict(max_iterations=9)),
                                      (28, dict(rho_min=0.0, t_min=0, refresh_period=1)), (35, dict(block_size=16))])
def test_scheduler_matches_the_oracle(handle, seed, kw):
    from paper_2606_08411_b200.scheduler import run_with_stub_model
    case = W.scheduler_case(seed, gen_len=192)
    cfg = dict(case["cfg"], **kw)
    r = S.run(cfg, case["base"], case["target"], case["gain"], case["prompt"])
    if r["min_margin"] <= 2e-5:
        pytest.skip(f"a decision within {r['min_margin']:.1e} of a threshold: not comparable across precisions")
    g = run_with_stub_model(handle, cfg, case["base"], case["target"], case["gain"], case["prompt"])
    compare(r, g)
    if "max_iterations" not in kw:
        assert g["output"].tolist() == case["target"][:case["eos_at"]].tolist()      # the decoded text itself


def test_scheduler_drives_refresh_and_attention(handle):
    """With device state: every refresh (Eq.12) scatters rows [0, L_refresh) of the recomputed states into the cache
    (bit copy; rows beyond the last L_refresh untouched) and every iteration runs the lane-batched attention of its
    active lanes (one group, per-lane prefix P + s) -- outputs finite, decoding unchanged."""
    from paper_2606_08411_b200 import binding as B
    from paper_2606_08411_b200.scheduler import run_with_stub_model
    case = W.scheduler_case(37, gen_len=192)
    cfg = case["cfg"]
    P, L, Wl = cfg["prompt_len"], cfg["gen_len"], cfg["lookahead"]
    Hq, Hkv, d, rows = 4, 2, 128, P + L + 8
    dev = torch.device("cuda:0")
    gen = torch.Generator(device=dev).manual_seed(5)
    rnd = lambda *s: torch.randn(*s, device=dev, generator=gen).bfloat16()
    k_cache, v_cache = rnd(Hkv, rows, d), rnd(Hkv, rows, d)
    k0, v0 = k_cache.clone(), v_cache.clone()
    k_src, v_src = rnd(P + L, Hkv, d), rnd(P + L, Hkv, d)
    max_rows = L + Wl
    q, k_new, v_new = rnd(max_rows, Hq, d), rnd(max_rows, Hkv, d), rnd(max_rows, Hkv, d)
    out = torch.zeros(max_rows, Hq, d, device=dev, dtype=torch.bfloat16)
    ds = B.al_sched_device_state(B.Handle.make_shape(Hq, Hkv, d, B.AL_BF16, rows), k_cache.data_ptr(), v_cache.data_ptr(),
                                 k_src.data_ptr(), v_src.data_ptr(), q.data_ptr(), k_new.data_ptr(), v_new.data_ptr(),
                                 out.data_ptr(), max_rows)
    r = S.run(cfg, case["base"], case["target"], case["gain"], case["prompt"])
    g = run_with_stub_model(handle, cfg, case["base"], case["target"], case["gain"], case["prompt"], device_state=ds)
    torch.cuda.synchronize()
    compare(r, g)
    last = r["refreshed"][-1]
    assert g["stats"]["refreshes"] == len(r["refreshed"]) and g["stats"]["refreshed_rows_last"] == last
    assert torch.equal(k_cache[:, :last], k_src[:last].permute(1, 0, 2)) and torch.equal(v_cache[:, :last], v_src[:last].permute(1, 0, 2))
    assert torch.equal(k_cache[:, last:], k0[:, last:]) and torch.equal(v_cache[:, last:], v0[:, last:])
    assert bool(torch.isfinite(out.float()).all()) and float(out.float().abs().max()) > 0


def test_scheduler_model_callback_and_errors(handle):
    """The model is a callback: a Python function wrapped as AL_MODEL_FN sees every iteration's lanes (host copies)
    and forwards to the stub kernel; a failing callback surfaces as AL_ERR_CUDA; a tree that outgrows max_tree as
    AL_ERR_UNSUPPORTED."""
    from paper_2606_08411_b200 import binding as B
    from paper_2606_08411_b200.scheduler import run_with_stub_model
    case = W.scheduler_case(21, gen_len=96)
    cfg = case["cfg"]
    lib = B.load_library()
    dev = torch.device("cuda:0")
    base_d = torch.from_numpy(case["base"]).to(dev); target_d = torch.from_numpy(case["target"]).to(dev)
    stub = B.al_stub_model(base_d.data_ptr(), target_d.data_ptr(), float(case["gain"]), cfg["vocab"])
    seen = []

    def model(user, lanes, steps, n_lanes, n_rows, row_pos, tokens, logits, stream):
        arr = np.ctypeslib.as_array(ctypes.cast(lanes, ctypes.POINTER(ctypes.c_int32)), shape=(n_lanes, 6))
        seen.append((n_lanes, n_rows, int(arr[:, 4].sum())))
        return lib.al_stub_model_fn(ctypes.addressof(stub), lanes, steps, n_lanes, n_rows, row_pos, tokens, logits, stream)

    lib.al_stub_model_fn.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_int32] * 2 + [ctypes.c_void_p] * 4
    fn = B.AL_MODEL_FN(model)
    r = S.run(cfg, case["base"], case["target"], case["gain"], case["prompt"])
    g = run_with_stub_model(handle, cfg, case["base"], case["target"], case["gain"], case["prompt"], model_fn=fn, model_user=None)
    compare(r, g)
    assert len(seen) == g["stats"]["model_calls"] and all(n_rows == q for _, n_rows, q in seen)
    bad = B.AL_MODEL_FN(lambda *a: 7)
    with pytest.raises(B.AlError) as e:
        run_with_stub_model(handle, cfg, case["base"], case["target"], case["gain"], case["prompt"], model_fn=bad)
    assert e.value.status == B.AL_ERR_CUDA
    with pytest.raises(B.AlError) as e:
        run_with_stub_model(handle, cfg, case["base"], case["target"], case["gain"], case["prompt"], max_tree=3)
    assert e.value.status == B.AL_ERR_UNSUPPORTED
