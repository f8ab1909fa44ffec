"""al_lm_head_confidence_static -- the LM head + transfer rule for callers that cannot allocate device memory: no
workspace argument, the per-(row, chunk) partials live in the library's file-scope device array (1 MiB).  Its
outputs must equal those of al_lm_head_confidence (same kernels, same plan: conf within the 2e-3 of the confidence
tests -- in fact bit-identical -- argmax / commit / tokens bit-exact), on two calls in a row of DIFFERENT shapes (the
array keeps the first call's contents and nothing is cleared), without a byte of device memory being allocated;
a shape whose partials do not fit is refused before anything is enqueued.

Collected last on purpose (pytest -x: a failure here hides no other test)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2606_08411_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handle():
    from paper_2606_08411_b200 import binding
    h = binding.Handle(0)
    yield h
    h.close()


def make_case(N, V, K, seed, dev):
    from paper_2606_08411_b200.step import to_device
    rng = np.random.default_rng(seed)
    hidden = W.round_to_bf16(rng.standard_normal((N, K)).astype(np.float32))
    weight = W.round_to_bf16((rng.standard_normal((V, K)) / np.sqrt(K)).astype(np.float32))
    hot = rng.integers(0, V, size=N)                       # half of the rows peaked on one token (conf near 1)
    pk = rng.random(N) < 0.5
    scale = 14.0 / np.maximum((weight[hot] ** 2).sum(1), 1e-6)
    hidden[pk] = W.round_to_bf16((weight[hot] * scale[:, None])[pk].astype(np.float32))
    tokens = np.where(rng.random(N) < 0.6, V - 1, 3).astype(np.int32)
    lanes = np.asarray([[0, 0, 0, 0, N // 2, 1], [0, 0, 0, N // 2, N - N // 2, 0]], np.int32)   # a refine lane: EOS suppressed
    return dict(N=N, V=V, K=K, hidden=to_device(hidden, "bf16", dev), weight=to_device(weight, "bf16", dev),
                tokens=torch.from_numpy(tokens).to(dev), lanes=torch.from_numpy(lanes).to(dev), eos=int(hot[0]))


def outputs(N, dev):
    return (torch.zeros(N, device=dev), torch.zeros(N, dtype=torch.int32, device=dev),
            torch.zeros(N, dtype=torch.uint8, device=dev), torch.zeros(N, dtype=torch.int32, device=dev))


def test_static_scratch_entry_matches_the_workspace_path_on_two_calls_in_a_row(handle):
    from paper_2606_08411_b200 import binding as B
    dev = torch.device("cuda:0")
    assert handle.al_lm_head_confidence_static_max_bytes() == 1 << 20
    cases = [make_case(300, 9000, 256, 71, dev), make_case(130, 5000, 136, 72, dev)]
    want = []
    for c in cases:                                         # the existing path, workspace poisoned
        ws = torch.full((handle.al_lm_head_confidence_workspace_bytes(c["N"], c["V"]),), 0xFF, dtype=torch.uint8, device=dev)
        o = outputs(c["N"], dev)
        handle.al_lm_head_confidence(c["hidden"], c["weight"], c["N"], c["V"], c["K"], c["tokens"], c["V"] - 1, c["eos"],
                                     0.9, c["lanes"], 2, B.AL_SELECT_FORCE_TOP1, *o, ws)
        want.append(o)
    got = [outputs(c["N"], dev) for c in cases]             # every buffer exists before the calls under test
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(dev), torch.cuda.mem_get_info(dev)[0]
    for c, o in zip(cases, got):                            # two calls in a row on the shared array, nothing cleared between
        handle.al_lm_head_confidence_static(c["hidden"], c["weight"], c["N"], c["V"], c["K"], c["tokens"], c["V"] - 1,
                                            c["eos"], 0.9, c["lanes"], 2, B.AL_SELECT_FORCE_TOP1, *o)
    torch.cuda.synchronize()
    after = torch.cuda.memory_allocated(dev), torch.cuda.mem_get_info(dev)[0]
    assert after[0] == before[0] and after[1] >= before[1], (before, after)      # no device memory was taken
    for c, g, w in zip(cases, got, want):
        assert float((g[0] - w[0]).abs().max()) <= 2e-3
        assert torch.equal(g[0], w[0])                      # same kernels, same plan: bit-identical
        assert torch.equal(g[1], w[1]) and torch.equal(g[2], w[2]) and torch.equal(g[3], w[3])
        assert int(g[2].sum()) > 0 and bool(torch.isfinite(g[0]).all())


def test_static_scratch_entry_refuses_what_does_not_fit(handle):
    from paper_2606_08411_b200 import binding as B
    dev = torch.device("cuda:0")
    N, V, K = 8192, 152064, 8                               # 2 MiB of partials: more than the array holds
    z = torch.zeros(8, dtype=torch.bfloat16, device=dev)    # never read: the call is refused before anything is enqueued
    o = outputs(8, dev)
    n0 = handle.al_launch_count
    with pytest.raises(B.AlError) as e:
        handle.al_lm_head_confidence_static(z, z, N, V, K, o[1], V - 1, -1, 0.9, None, 0, 0, *o)
    assert e.value.status == B.AL_ERR_UNSUPPORTED and "static array" in str(e.value)
    assert handle.al_launch_count == n0
