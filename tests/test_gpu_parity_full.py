"""GPU parity at the sizes bench.py times (BASELINE configs[3], configs[4]) and on the paths the smaller
cases never reach: EVERY output element against the CPU oracle, in the launch configuration of bench.py
(al_lane_plan once, al_lane_attention_planned per layer; layer-batched refresh; one confidence launch).

Tolerances are those of tests/test_gpu_parity.py (BASELINE.json north_star).
"""
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


@pytest.fixture(scope="module")
def cfg5():
    return W.cfg5_throughput_batch()


@pytest.fixture(scope="module")
def cfg4():
    return W.cfg4_long_llada()          # all 32 layers, as bench.py runs it


def make_step(handle, wl, **kw):
    from paper_2606_08411_b200.step import LaneStep
    return LaneStep(handle, wl, **kw)


def to_np(t):
    return t.detach().float().cpu().numpy() if t.dtype in (torch.bfloat16, torch.float32) else t.detach().cpu().numpy()


def attention_all_rows(wl, out, lse, layers):
    """max normwise relative error (reading C10) and max LSE error over ALL rows and heads of `layers`."""
    worst, worst_lse = 0.0, 0.0
    for layer in layers:
        ref, ref_lse = oracle.lane_attention(wl.q[layer], wl.k_new[layer], wl.v_new[layer], wl.k_cache[layer],
                                             wl.v_cache[layer], wl.lanes)
        o = out[layer]
        assert np.isfinite(o).all()
        err = np.abs(o - ref).max(axis=-1) / np.maximum(np.abs(ref).max(axis=-1), 1e-30)
        worst = max(worst, float(err.max()))
        worst_lse = max(worst_lse, float(np.abs(lse[layer] - ref_lse).max()))
    return worst, worst_lse


def confidence_all_rows(handle, wl, st=None):
    st = st or make_step(handle, wl)
    st.confidence(); torch.cuda.synchronize()
    ref = oracle.confidence_select(wl.logits, wl.tokens, wl.mask_id, wl.eos_id, wl.threshold, wl.lanes)
    conf, am, commit, tok = to_np(st.conf), to_np(st.argmax), to_np(st.commit), to_np(st.tokens_out)
    assert np.abs(conf - ref["conf"]).max() <= 2e-3
    assert np.array_equal(am, ref["argmax"])                     # first maximiser everywhere (reading C6)
    tau_ok = np.abs(ref["conf"] - wl.threshold) > 4e-3
    sel = tau_ok & ((ref["conf"] - ref["p2"]) > 1e-3)
    assert np.array_equal(commit[tau_ok], ref["commit"][tau_ok])
    assert np.array_equal(tok[sel], ref["tokens_out"][sel])
    assert (~tau_ok).mean() <= 0.08
    return st, ref


def refresh_all_bytes(handle, wl, st=None):
    st = st or make_step(handle, wl)
    bits = (lambda t: t.view(torch.int16)) if wl.dtype == "bf16" else (lambda t: t)
    ek, ev = bits(st.k_cache).cpu().numpy().copy(), bits(st.v_cache).cpu().numpy().copy()
    st.refresh(); torch.cuda.synchronize()
    oracle.kv_refresh(ek, ev, np.ascontiguousarray(bits(st.k_src).cpu().numpy()),
                      np.ascontiguousarray(bits(st.v_src).cpu().numpy()), wl.refresh_pos, wl.refresh_base_row)
    assert np.array_equal(bits(st.k_cache).cpu().numpy(), ek)
    assert np.array_equal(bits(st.v_cache).cpu().numpy(), ev)


# ------------------------------------------------------------------------------------------------
# BASELINE configs[4]: the workload bench.py times by default
# ------------------------------------------------------------------------------------------------
def test_cfg5_attention_every_row_every_head(handle, cfg5):
    """All 3264 x 28 outputs of the stream-K launch (148 CTAs, every one ending in a two-partial merge)."""
    st = make_step(handle, cfg5)
    handle.al_validate_lanes(st.shape, st.lanes, cfg5.n_lanes, cfg5.total_q_rows)
    st.attention(); torch.cuda.synchronize()
    worst, worst_lse = attention_all_rows(cfg5, to_np(st.out), to_np(st.lse), [0])
    assert worst <= 1e-2, worst
    assert worst_lse <= 1e-3, worst_lse


def test_cfg5_confidence_every_row(handle, cfg5):
    """3264 x 152064: cluster size 1, one CTA per full-vocabulary row."""
    confidence_all_rows(handle, cfg5)


def test_cfg5_refresh_absolute_pool_rows(handle, cfg5):
    st = make_step(handle, cfg5)
    handle.al_validate_refresh(st.shape, st.pos, int(st.pos.numel()), cfg5.refresh_base_row)
    refresh_all_bytes(handle, cfg5, st)


# ------------------------------------------------------------------------------------------------
# BASELINE configs[3]: 32 layers resident
# ------------------------------------------------------------------------------------------------
def test_cfg4_attention_every_row_first_and_last_layer(handle, cfg4):
    st = make_step(handle, cfg4)
    st.attention(); torch.cuda.synchronize()
    layers = [0, cfg4.n_layers - 1]
    out = {l: to_np(st.out[l]) for l in layers}
    lse = {l: to_np(st.lse[l]) for l in layers}
    worst, worst_lse = attention_all_rows(cfg4, out, lse, layers)
    assert worst <= 1e-2, worst
    assert worst_lse <= 1e-3, worst_lse
    # every layer ran (the plan is reused 32 times): no layer's output is left at its zero fill
    assert bool((st.out.float().abs().amax(dim=(1, 2, 3)) > 0).all())


def test_cfg4_confidence_and_layer_batched_refresh(handle, cfg4):
    st = make_step(handle, cfg4, want_lse=False)
    confidence_all_rows(handle, cfg4, st)                  # 384 x 126464
    refresh_all_bytes(handle, cfg4, st)                    # 320 rows x 32 layers in one launch


# ------------------------------------------------------------------------------------------------
# confidence: the 8-CTA cluster path (one row split over eight CTAs, merged through DSMEM)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_rows,vocab", [(32, W.DREAM_VOCAB), (64, 131072)])
def test_confidence_cluster_of_eight(handle, n_rows, vocab):
    """N <= 74 rows over a >= 131072-wide bf16 vocabulary is the paper's own operating point (one lane of 32
    rows, batch 1: PAPER.md L197) and the only shape that takes cluster size 8.  Planted: exact ties whose
    two maximisers sit in DIFFERENT cluster ranks (lower index must win), a maximum in the last rank's
    last element, and a refine lane whose EOS logit is the row maximum (suppressed)."""
    rng = np.random.default_rng(800 + n_rows)
    x = (rng.standard_normal((n_rows, vocab), dtype=np.float32) * np.float32(3.0))
    chunk = vocab // 8
    eos = 5 * chunk + 17
    x[0, 2 * chunk + 5] = 40.0; x[0, 6 * chunk + 9] = 40.0            # tie across ranks 2 and 6
    x[1, chunk - 1] = 33.0; x[1, chunk] = 33.0                         # tie across the rank 0 / 1 border
    x[2, vocab - 1] = 35.0                                             # last element of the last rank
    x[3, eos] = 50.0; x[3, 11] = 30.0                                  # refine lane: EOS suppressed, 11 wins
    x[20, eos] = 50.0                                                  # generate lane: EOS stands
    x = W.round_to_bf16(x)
    lanes = np.array([[0, 0, 0, 0, 16, W.LANE_FLAG_REFINE], [0, 0, 0, 16, n_rows - 16, 0]], np.int32)
    tokens = np.full(n_rows, 7, np.int32); tokens[::3] = 3
    wl = W.cfg1_tiny()
    wl.dtype = "bf16"; wl.logits = x; wl.tokens = tokens; wl.mask_id = 7; wl.eos_id = eos; wl.lanes = lanes
    wl.threshold = 0.9
    st, ref = confidence_all_rows(handle, wl)
    am = to_np(st.argmax)
    assert [int(am[0]), int(am[1]), int(am[2]), int(am[3]), int(am[20])] == [2 * chunk + 5, chunk - 1, vocab - 1, 11, eos]
    assert to_np(st.conf)[0] == pytest.approx(0.5, abs=2e-3)


# ------------------------------------------------------------------------------------------------
# al_lane_step_host: the e2e entry point of bench.py
# ------------------------------------------------------------------------------------------------
def check_step_host(handle, wl):
    from paper_2606_08411_b200.step import HostStep, to_device
    dev = torch.device("cuda:0")
    hstep = HostStep(handle, wl, device=dev)
    k_cache, v_cache = to_device(wl.k_cache, wl.dtype, dev), to_device(wl.v_cache, wl.dtype, dev)
    hstep.out.zero_(); hstep.conf.zero_()
    hstep.run(k_cache, v_cache); torch.cuda.synchronize()
    tol = 1e-2 if wl.dtype == "bf16" else 2e-5
    covered = np.zeros(wl.total_q_rows, bool)
    for l in wl.lanes:
        covered[l[W.LANE_Q_START]:l[W.LANE_Q_START] + l[W.LANE_Q_LEN]] = True
    out = hstep.out.float().numpy()
    for layer in range(wl.n_layers):                       # attention saw the cache BEFORE the refresh (C16)
        ref, _ = oracle.lane_attention(wl.q[layer], wl.k_new[layer], wl.v_new[layer], wl.k_cache[layer],
                                       wl.v_cache[layer], wl.lanes)
        err = np.abs(out[layer][covered] - ref[covered]).max(-1) / np.abs(ref[covered]).max(-1)
        assert err.max() <= tol, (layer, err.max())
    r = oracle.confidence_select(wl.logits, wl.tokens, wl.mask_id, wl.eos_id, wl.threshold, wl.lanes)
    assert np.abs(hstep.conf.numpy() - r["conf"]).max() <= 2e-3
    assert np.array_equal(hstep.argmax.numpy(), r["argmax"])
    tau_ok = np.abs(r["conf"] - wl.threshold) > 4e-3
    sel = tau_ok & ((r["conf"] - r["p2"]) > 1e-3)
    assert np.array_equal(hstep.commit.numpy()[tau_ok], r["commit"][tau_ok])
    assert np.array_equal(hstep.tokens_out.numpy()[sel], r["tokens_out"][sel])
    kc, vc = wl.k_cache.copy(), wl.v_cache.copy()           # the refreshed cache, bit for bit
    oracle.kv_refresh(kc, vc, wl.k_src, wl.v_src, wl.refresh_pos, wl.refresh_base_row)
    assert np.array_equal(k_cache.float().cpu().numpy(), kc)
    assert np.array_equal(v_cache.float().cpu().numpy(), vc)
    assert hstep.h2d_bytes > 0 and hstep.d2h_bytes >= out.nbytes // (2 if wl.dtype == "bf16" else 1)


def test_step_host_ragged_and_cfg2(handle):
    check_step_host(handle, W.ragged_case(451))
    check_step_host(handle, W.cfg2_llada_layer())
    check_step_host(handle, W.cfg1_tiny())                  # fp32: the plain-ALU attention path, no plan


def test_step_host_all_layers(handle):
    """n_layers > 1: one plan, one attention launch per layer on that layer's cache, one layer-batched refresh."""
    check_step_host(handle, W.cfg4_long_llada(n_layers=3))


def test_step_host_validates_before_anything_is_enqueued(handle):
    from paper_2606_08411_b200 import binding as B
    from paper_2606_08411_b200.step import HostStep, to_device
    wl = W.ragged_case(452)
    dev = torch.device("cuda:0")
    hstep = HostStep(handle, wl, device=dev)
    k_cache, v_cache = to_device(wl.k_cache, wl.dtype, dev), to_device(wl.v_cache, wl.dtype, dev)
    before_k = k_cache.clone()
    hstep.out.fill_(7.0)
    launches = handle.al_launch_count
    hstep.hs.eos_id = wl.vocab + 5                          # only the LAST part (confidence) is invalid
    with pytest.raises(B.AlError) as e:
        hstep.run(k_cache, v_cache)
    torch.cuda.synchronize()
    assert e.value.status == B.AL_ERR_INVALID_ARG
    assert handle.al_launch_count == launches               # no kernel was enqueued ...
    assert bool((hstep.out.float() == 7.0).all())           # ... no result copied back ...
    assert torch.equal(k_cache, before_k)                   # ... and the cache was not refreshed


# ------------------------------------------------------------------------------------------------
# rows no lane may see can hold anything (include/asynclane.h, finite-input contract)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [461, 462, 463])
def test_attention_ignores_nan_in_cache_rows_no_lane_sees(handle, seed):
    """Cache rows outside every lane's visible range are poisoned with NaN / Inf (unwritten or recycled
    memory in a serving cache).  The oracle never reads them; the kernel multiplies them by exact zeros
    only after zeroing what the last key tile rounds up to -- the output must be bit-identical."""
    wl = W.ragged_case(seed)
    st = make_step(handle, wl)
    st.attention(); torch.cuda.synchronize()
    clean, clean_lse = st.out.clone(), st.lse.clone()
    seen = np.zeros(wl.cache_rows, bool)
    for l in wl.lanes:
        seen[l[W.LANE_KV_BASE_ROW]:l[W.LANE_KV_BASE_ROW] + l[W.LANE_PREFIX_LEN]] = True
    hidden = torch.from_numpy(~seen).to(st.device)
    assert int(hidden.sum()) > 0
    st.k_cache[:, :, hidden] = float("nan")
    st.v_cache[:, :, hidden] = float("inf") if seed % 2 else float("nan")
    st.out.zero_()
    st.attention(); torch.cuda.synchronize()
    assert bool(torch.isfinite(st.out.float()).all())
    assert torch.equal(st.out, clean) and torch.equal(st.lse, clean_lse)


def test_validate_refresh_rejects_duplicates_and_out_of_range(handle):
    from paper_2606_08411_b200 import binding as B
    wl = W.cfg1_tiny()
    st = make_step(handle, wl)
    handle.al_validate_refresh(st.shape, st.pos, int(st.pos.numel()), wl.refresh_base_row)
    dev = st.device
    for bad in ([3, 3, 9], [9, 3], [0, wl.cache_rows], [-1, 2]):
        pos = torch.tensor(bad, dtype=torch.int32, device=dev)
        with pytest.raises(B.AlError) as e:
            handle.al_validate_refresh(st.shape, pos, len(bad), 0)
        assert e.value.status == B.AL_ERR_INVALID_ARG
    with pytest.raises(B.AlError):                           # in range only without the base offset
        handle.al_validate_refresh(st.shape, torch.tensor([wl.cache_rows - 1], dtype=torch.int32, device=dev), 1, 1)
    handle.al_validate_refresh(st.shape, st.pos, 0, 0)       # empty list: valid
