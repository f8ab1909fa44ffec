#!/usr/bin/env python
"""bench.py -- the lane-batched denoising step of AsyncLane on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is ONE pass of the whole hot path (lane attention for every layer of the
workload, compact KV refresh, confidence/argmax/threshold select) over one batch of seeded
synthetic input.  The default workload is BASELINE.json configs[4] (16 Dream-shaped sequences), the
largest single-GPU configuration; configs[1..3] are measured in the same run with fewer steps and
reported under the extra key `workloads` (step time, per-part time and roofline fraction).

What is timed:
  value     K steps, inputs resident in HBM, each step one CUDA-graph replay; consecutive steps run
            on DISTINCT copies of every streamed buffer (rotation set > 2x L2) so nothing is served
            from L2.  Device time from CUDA events on the launching stream, max over ranks.
  roofline  per-part device time: every part (attention = plan + all layers, refresh, confidence) has
            a graph of its own that runs it on every resident copy in turn, replayed right after the
            timed region and timed with CUDA events on the stream (time / launches in the graph).
  e2e       the same step through the C-ABI host entry al_lane_step_host: every step copies its
            inputs from pinned host memory, runs the kernels and copies the results back.
  cpu_baseline / --impl reference   the CPU oracle (oracle/, fp64, as it stands) on the host cores.

Multi-GPU: the path does not shard (BASELINE north_star: one GPU, no collectives) -> "replicas
only": every rank runs an independent replica, value = all ranks' tokens / max-over-ranks time.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_BYTES = 126e6
METRIC = "lane-step query tok/s (parts: attention TFLOP/s, refresh+confidence GB/s vs peak)"
UNIT = "query tok/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=float(p["hbm_gbs"]), tensor=float(p["bf16_tflops"]),
                    tensor_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    # fallback stated by /opt/skills/guides/B200_PROFILING.md
    return dict(hbm=6650.0, tensor=1590.0, tensor_sustained=1400.0, source="fallback")


def load_traffic(workload: str):
    """dram bytes per launch from the committed ncu --set full capture (profiles/), if any."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if os.path.exists(path):
        try:
            return json.load(open(path)).get(workload, {})
        except Exception:
            return {}
    return {}


# --------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed regions run."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period_s: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reason_bits, self.power = [], 0, []
        self.active = threading.Event()
        self.stop_flag = threading.Event()
        self.ok = False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag.is_set():
            if self.active.is_set():
                try:
                    self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                    try:
                        r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev))
                    except Exception:
                        r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev))
                    self.reason_bits |= r
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.dev) / 1000.0)
                except Exception:
                    pass
            time.sleep(self.period)

    def reset(self):
        self.samples, self.reason_bits, self.power = [], 0, []

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unsampled"], "samples": 0}
        s = sorted(self.samples)
        reasons = [n for b, n in self.REASONS.items() if (self.reason_bits & b) and n != "gpu_idle"]
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(s), "power_w_max": round(max(self.power), 1) if self.power else None}


# --------------------------------------------------------------------------------------------------
def max_over_ranks(ms: float, dist, device) -> float:
    """Replicas only: every rank times its own replica on its own device; the job's step time is the
    slowest rank's (one all_reduce(MAX) of a scalar -- the only collective, and it is not on the data path)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, step_ms: float) -> float:
    """Aggregate throughput of `world` independent replicas: all ranks' units over the slowest rank's time."""
    return world * units_per_rank / (step_ms * 1e-3)


# --------------------------------------------------------------------------------------------------
def oracle_step(oracle, wl, lanes, rows):
    """One pass of the hot path on the CPU oracle over whole lanes `lanes` / logits rows `rows`."""
    for layer in range(wl.n_layers):
        oracle.lane_attention(wl.q[layer], wl.k_new[layer], wl.v_new[layer], wl.k_cache[layer], wl.v_cache[layer],
                              lanes)
    kc, vc = wl.k_cache, wl.v_cache            # in place: the oracle's refresh is idempotent
    oracle.kv_refresh(kc, vc, wl.k_src, wl.v_src, wl.refresh_pos, wl.refresh_base_row)
    r0, r1 = (int(rows.min()), int(rows.max()) + 1) if len(rows) else (0, 0)     # dense: a view, no copy
    oracle.confidence_select(wl.logits[r0:r1], wl.tokens[r0:r1], wl.mask_id, wl.eos_id, wl.threshold, None)


def time_oracle(wl, steps: int, warmup: int, budget_s: float):
    """Times the oracle on a bounded sample: the first n whole lanes (lanes are independent)
    and the logits rows of those lanes, n chosen so that steps+warmup passes fit in `budget_s`."""
    import numpy as np
    import oracle
    from paper_2606_08411_b200 import workloads as W
    oracle.build()
    cores = oracle.num_threads()
    one = wl.lanes[:1]
    rows1 = np.arange(int(one[0, W.LANE_Q_START]), int(one[0, W.LANE_Q_START] + one[0, W.LANE_Q_LEN]))
    rows1 = rows1[rows1 < wl.logits.shape[0]]
    oracle_step(oracle, wl, one, rows1)                       # page-in, thread pool start
    t0 = time.perf_counter()
    oracle_step(oracle, wl, one, rows1)
    t_lane = max(time.perf_counter() - t0, 1e-4)
    n = int(max(1, min(wl.n_lanes, (budget_s / max(1, steps + warmup)) / t_lane)))
    lanes = wl.lanes[:n]
    rows = np.concatenate([np.arange(int(l[W.LANE_Q_START]), int(l[W.LANE_Q_START] + l[W.LANE_Q_LEN])) for l in lanes])
    rows = rows[rows < wl.logits.shape[0]]
    tokens = int(lanes[:, W.LANE_Q_LEN].sum())
    for _ in range(warmup):
        oracle_step(oracle, wl, lanes, rows)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(oracle, wl, lanes, rows)
    dt = time.perf_counter() - t0
    sample = (f"{n} of {wl.n_lanes} whole lanes ({tokens} of {wl.total_q_rows} query rows; all heads, all "
              f"{wl.n_layers} layer(s)) + their {rows.size} logits rows + the full refresh, {steps} passes")
    return dict(value=tokens * steps / dt, unit=UNIT, cores=cores, kind="oracle", sample=sample), dt / steps


# --------------------------------------------------------------------------------------------------
def run_reference(args, rank: int):
    if rank != 0:
        return
    from paper_2606_08411_b200 import workloads as W
    wl = W.CONFIGS[args.workload]()
    cpu, s_per_step = time_oracle(wl, args.steps, args.warmup, budget_s=150.0)
    line = {"impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl.name, "note": "CPU oracle (oracle/) on the host cores"},
            "cpu_baseline": cpu,
            "e2e": {"value": cpu["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
def part_rooflines(wl, acc, part_ms, step_ms, peaks, traffic):
    """Roofline of every part from its own device time (algorithmic numerators of accounting.py)."""
    parts = {}
    ai = acc["attn_flops"] / acc["attn_bytes"]
    ridge = peaks["tensor"] * 1e12 / (peaks["hbm"] * 1e9)
    ta, tr, tc = (part_ms[k] * 1e-3 for k in ("attention", "refresh", "confidence"))
    if ai < ridge:
        parts["attention"] = dict(bound="hbm", achieved=acc["attn_bytes"] / ta / 1e9, peak=peaks["hbm"], unit="GB/s")
    else:
        parts["attention"] = dict(bound="tensor", achieved=acc["attn_flops"] / ta / 1e12, peak=peaks["tensor"],
                                  unit="TFLOP/s")
    parts["attention"].update(ms=ta * 1e3, launches=wl.n_layers, tflops=acc["attn_flops"] / ta / 1e12,
                              gbs=acc["attn_bytes"] / ta / 1e9, arithmetic_intensity=ai,
                              note="time of al_lane_plan (1 launch) + al_lane_attention_planned (1 launch per layer)")
    parts["refresh"] = dict(bound="hbm", achieved=acc["refresh_bytes"] / tr / 1e9, peak=peaks["hbm"], unit="GB/s",
                            ms=tr * 1e3, launches=1)
    parts["confidence"] = dict(bound="hbm", achieved=acc["confidence_bytes"] / tc / 1e9, peak=peaks["hbm"],
                               unit="GB/s", ms=tc * 1e3, launches=1)
    for k, p in parts.items():
        p["frac"] = p["achieved"] / p["peak"]
        if p["bound"] == "hbm" and p["frac"] > 1.0:      # the measured peak is a COPY (read + write); a read-only stream can pass it
            p["note"] = "read-only stream above the measured copy bandwidth (read+write figure)"
        p["traffic"] = traffic.get(k)
        p["share_of_step"] = p["ms"] / step_ms
    return parts


def measure_resident(h, wl, dev, stream, dist, sampler, steps, warmup, kernel_events=True):
    """`steps` timed replays of the whole-step CUDA graph over rotating resident copies of `wl`, then the
    per-part times on the parts' own graphs.  Returns the copies too (the e2e leg reuses their caches)."""
    import torch
    from paper_2606_08411_b200.step import LaneStep

    first = LaneStep(h, wl, device=dev, want_lse=False)
    per_copy = first.streamed_bytes()
    n_copies = max(2, int(math.ceil(2.2 * L2_BYTES / per_copy)))
    copies = [first] + [first.replicate() for _ in range(n_copies - 1)]
    graphs, part_graphs = [], []
    launches_per_step = None
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        copies[0].run(stream)                                  # load modules / set attributes before capture
        stream.synchronize()
        for st in copies:
            g = torch.cuda.CUDAGraph()                         # the step as a user runs it: kernels only
            before = h.al_launch_count
            with torch.cuda.graph(g, stream=stream):
                st.run(stream)
            launches_per_step = h.al_launch_count - before
            graphs.append(g)
        # Per-part times: ONE graph per part that runs the part on every resident copy in turn (at least 4
        # launches), so that consecutive launches never share data through L2 and the time between two
        # launches inside the graph is what a step sees (event nodes inside the step graph would cost a few us
        # and break the programmatic-dependent-launch edges; one graph replay per launch would add the graph
        # launch latency, ~2 us, to every sample)
        if kernel_events:
            inner = max(n_copies, 4)
            for name in ("attention", "refresh", "confidence"):
                gp = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gp, stream=stream):
                    for i in range(inner):
                        getattr(copies[i % n_copies], name)(stream)
                part_graphs.append((name, gp, inner))
    stream.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up, then EXACTLY `steps` timed steps ---------------------------------------------
    with torch.cuda.stream(stream):
        for i in range(warmup):
            graphs[i % n_copies].replay()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.active.set()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in range(steps):
            graphs[i % n_copies].replay()
        e1.record(stream)
    barrier()
    sampler.active.clear()
    step_ms = e0.elapsed_time(e1) / steps

    # per-part device times: right after the timed region, every part's own graph is replayed over the
    # same rotation of copies (so its inputs come from HBM, not L2) and timed with CUDA events on the stream
    part_ms = None
    if kernel_events:
        part_ms = {}
        sampler.active.set()
        for name, gp, inner in part_graphs:
            reps = max(40 // inner, 8)
            with torch.cuda.stream(stream):
                gp.replay()
                e0.record(stream)
                for i in range(reps):
                    gp.replay()
                e1.record(stream)
            barrier()
            part_ms[name] = e0.elapsed_time(e1) / (reps * inner)
            part_ms["n_samples"] = reps * inner
        sampler.active.clear()
    # warm-L2 step (cold and warm reported separately): the same graph replayed on ONE copy, for
    # workloads whose streamed bytes fit the L2 at all -- not the headline, which always rotates the copies
    warm_ms = None
    if kernel_events and per_copy <= L2_BYTES:
        n_warm = max(20, min(steps, 200))
        with torch.cuda.stream(stream):
            for _ in range(5):
                graphs[0].replay()
            e0.record(stream)
            for _ in range(n_warm):
                graphs[0].replay()
            e1.record(stream)
        barrier()
        warm_ms = e0.elapsed_time(e1) / n_warm
    return dict(step_ms=step_ms, part_ms=part_ms, launches_per_step=launches_per_step, copies=copies,
                n_copies=n_copies, per_copy=per_copy, barrier=barrier, graphs=graphs, part_graphs=part_graphs,
                warm_ms=warm_ms)


def measure_next_rows(h, dev, stream, peaks):
    """SURVEY 8(f) rows, each timed on its own (CUDA events on the stream, inputs resident): the fused LM head at the
    LLaDA-layer and batch-16 shapes (next to the library route it replaces: cuBLAS GEMM + al_confidence_select on
    materialised bf16 logits), al_lane_status on the batch-16 lanes, the Eq.12 refresh forward of one Dream-shaped
    sequence, the compact refresh on a random sorted subset and on a contiguous run (reading C8), and Algorithm 1 end to
    end with the table-driven stub model."""
    import numpy as np
    import torch
    from paper_2606_08411_b200 import binding as B, workloads as W
    from paper_2606_08411_b200.scheduler import run_with_stub_model

    def timed(fn, n):
        torch.cuda.synchronize()                 # the inputs were made on the default stream: nothing else may be running
        with torch.cuda.stream(stream):
            fn(); fn()
            stream.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(n):
                fn()
            e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    def timed_graph(fn, n, inner=8):
        """us per call with `inner` calls captured into one CUDA graph (as the steps are timed: no host launch cost)"""
        g = torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.stream(stream):
            fn()
            stream.synchronize()
            with torch.cuda.graph(g, stream=stream):
                for _ in range(inner):
                    fn()
        return timed(lambda: g.replay(), n) / inner

    out = {}
    gen = torch.Generator(device=dev).manual_seed(1)
    rnd = lambda *sh: torch.randn(*sh, device=dev, generator=gen)
    for name, N, V, K in (("llada_layer_128x126464x4096", 128, W.LLADA_VOCAB, 4096),
                          ("batch16_3264x152064x3584", 3264, W.DREAM_VOCAB, 3584)):
        hid = rnd(N, K).bfloat16()
        wts = [(rnd(V, K) / K ** 0.5).bfloat16() for _ in range(2)]         # two copies: 2 x 1 GB > L2
        tok = torch.zeros(N, dtype=torch.int32, device=dev)
        conf = torch.zeros(N, device=dev); am = torch.zeros(N, dtype=torch.int32, device=dev)
        cm = torch.zeros(N, dtype=torch.uint8, device=dev); to = torch.zeros(N, dtype=torch.int32, device=dev)
        ws = torch.empty(h.al_lm_head_confidence_workspace_bytes(N, V), dtype=torch.uint8, device=dev)
        logits = torch.empty(N, V, device=dev, dtype=torch.bfloat16)
        i = [0]

        def fused():
            i[0] += 1
            h.al_lm_head_confidence(hid, wts[i[0] & 1], N, V, K, tok, 7, -1, 0.9, None, 0, 0, conf, am, cm, to, ws, stream)

        def library():
            i[0] += 1
            torch.matmul(hid, wts[i[0] & 1].t(), out=logits)
            h.al_confidence_select(logits, N, V, V, tok, 7, -1, 0.9, None, 0, 0, conf, am, cm, to, None, stream)

        tf, tl = timed(fused, 10), timed(library, 10)
        flops = 2.0 * N * V * K
        out["lm_head_fused_" + name] = {"us": tf, "tflops": flops / tf / 1e6, "frac_of_bf16_peak": flops / tf / 1e6 / peaks["tensor"],
                                        "weight_gbs": V * K * 2 / tf / 1e3, "frac_of_hbm_peak": V * K * 2 / tf / 1e3 / peaks["hbm"],
                                        "library_route_us": tl, "library_route": "torch.matmul (cuBLAS) -> bf16 logits -> al_confidence_select"}
        del wts, logits, hid
        torch.cuda.empty_cache()
    # lane status on the batch-16 lanes (102 lanes, 3264 rows)
    wl_lanes = W.make_lanes(W.cfg5_lane_tree(np.random.default_rng(W.SEED_BASE + 5), 16, 1280))
    n_l, n_r = len(wl_lanes), int(wl_lanes[:, W.LANE_Q_LEN].sum())
    lanes_d = torch.from_numpy(wl_lanes).to(dev)
    ti = torch.full((n_r,), 7, dtype=torch.int32, device=dev); cf = torch.rand(n_r, device=dev, generator=gen)
    am = torch.randint(0, 100, (n_r,), dtype=torch.int32, device=dev)
    cm = torch.zeros(n_r, dtype=torch.uint8, device=dev); to = ti.clone() + 1
    stt = torch.zeros((n_l, 8), dtype=torch.int32, device=dev)
    dl = torch.tensor([13, 30], dtype=torch.int32, device=dev)
    f_status = lambda: h.al_lane_status(lanes_d, n_l, n_r, ti, cf, am, 7, 2, 0.9, dl, None, cm, to, stt, stream)
    out["lane_status_batch16"] = {"us": timed_graph(f_status, 20), "us_direct_launch": timed(f_status, 50), "lanes": n_l, "rows": n_r}
    # refresh forward (Eq.12) of one Dream-shaped sequence: L_refresh = 1024, 28q / 4kv heads, d = 128
    Lr, Hq, Hkv, d = 1024, 28, 4, 128
    shape = B.Handle.make_shape(Hq, Hkv, d, B.AL_BF16, Lr + 64)
    q, k, v = rnd(Lr, Hq, d).bfloat16(), rnd(Lr, Hkv, d).bfloat16(), rnd(Lr, Hkv, d).bfloat16()
    kc, vc = rnd(Hkv, Lr + 64, d).bfloat16(), rnd(Hkv, Lr + 64, d).bfloat16()
    o = torch.zeros_like(q)
    ln = torch.tensor([[0, 0, 0, 0, Lr, 0]], dtype=torch.int32, device=dev)
    wsa = torch.empty(h.al_lane_attention_workspace_bytes(shape, 1, Lr, 0), dtype=torch.uint8, device=dev)
    f_rf = lambda: h.al_refresh_forward(shape, q, k, v, kc, vc, ln, 1, Lr, 0, o, None, wsa, stream)
    t_rf = timed_graph(f_rf, 20, inner=4)
    fl = 4.0 * Hq * d * Lr * Lr
    out["refresh_forward_dream_1024"] = {"us": t_rf, "us_direct_launch": timed(f_rf, 30), "tflops": fl / t_rf / 1e6,
                                         "frac_of_bf16_peak": fl / t_rf / 1e6 / peaks["tensor"],
                                         "note": "plan + attention + append, 4 calls per CUDA-graph replay; the direct-launch figure includes the host's tensor-map encoding"}
    # compact refresh, both position sets of reading C8: a sorted random subset of the prefix (what the
    # workloads use) and the contiguous run [0, R) of Eq.12 -- config-4 shape: 32 layers, 320 of 1280 rows, 32 kv-heads.
    # Two cache sets (2 x 0.8 GB) alternate so that no launch finds its rows in L2.
    Lc, Hc, R, rows_c = 32, 32, 320, 1536
    shape_r = B.Handle.make_shape(32, Hc, 128, B.AL_BF16, rows_c)
    caches = [(torch.zeros(Lc, Hc, rows_c, 128, device=dev, dtype=torch.bfloat16), torch.zeros(Lc, Hc, rows_c, 128, device=dev, dtype=torch.bfloat16)) for _ in range(2)]
    srcs = [(rnd(Lc, R, Hc, 128).bfloat16(), rnd(Lc, R, Hc, 128).bfloat16()) for _ in range(2)]
    rngr = np.random.default_rng(20260608)
    pos_sets = {"random_sorted": np.sort(rngr.choice(1280, size=R, replace=False)).astype(np.int32), "contiguous": np.arange(R, dtype=np.int32)}
    rbytes = 2 * 2 * R * Hc * 128 * 2 * Lc + 4 * R
    for nm, pos in pos_sets.items():
        pd = torch.from_numpy(pos).to(dev)
        state = {"i": 0}
        def one():
            i = state["i"] = state["i"] ^ 1
            h.al_kv_refresh(shape_r, caches[i][0], caches[i][1], srcs[i][0], srcs[i][1], pd, R, 0, Lc, Hc * rows_c * 128, R * Hc * 128, stream)
        t = timed(one, 40)
        out["refresh_cfg4_shape_" + nm] = {"us": t, "gbs": rbytes / t / 1e3, "frac_of_hbm_peak": rbytes / t / 1e3 / peaks["hbm"]}
    del caches, srcs
    # launch floor: the smallest launch of this library -- al_kv_refresh of ONE row, one CTA --
    # back to back inside a CUDA graph, as the steps are timed: what a kernel of a single-layer step costs at least
    pd1 = torch.zeros(1, dtype=torch.int32, device=dev)
    kc1, vc1 = torch.zeros(Hkv, 8, d, device=dev, dtype=torch.bfloat16), torch.zeros(Hkv, 8, d, device=dev, dtype=torch.bfloat16)
    ks1, vs1 = torch.zeros(1, Hkv, d, device=dev, dtype=torch.bfloat16), torch.zeros(1, Hkv, d, device=dev, dtype=torch.bfloat16)
    shape1 = B.Handle.make_shape(Hq, Hkv, d, B.AL_BF16, 8)
    gfl = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        h.al_kv_refresh(shape1, kc1, vc1, ks1, vs1, pd1, 1, 0, 1, 0, 0, stream)
        stream.synchronize()
        with torch.cuda.graph(gfl, stream=stream):
            for _ in range(20):
                h.al_kv_refresh(shape1, kc1, vc1, ks1, vs1, pd1, 1, 0, 1, 0, 0, stream)
    out["launch_floor"] = {"us_per_launch": timed(lambda: gfl.replay(), 20) / 20,
                           "what": "al_kv_refresh of one row (one CTA), 20 launches per CUDA-graph replay"}
    # Algorithm 1 with the stub model (whole decode of 192 tokens, one synchronisation per iteration)
    case = W.scheduler_case(37, gen_len=192)
    t0 = time.perf_counter()
    reps = 5
    for _ in range(reps):
        r = run_with_stub_model(h, case["cfg"], case["base"], case["target"], case["gain"], case["prompt"])
    dt = (time.perf_counter() - t0) / reps
    out["scheduler_stub_model_192"] = {"ms_per_decode": dt * 1e3, "iterations": r["stats"]["iterations"],
                                       "us_per_iteration": dt * 1e6 / max(1, r["stats"]["iterations"]),
                                       "decoded_tokens": int(len(r["output"])), "forks": r["stats"]["forks"],
                                       "note": "stub model: measures the scheduler's per-iteration overhead (H2D, 4 kernels, D2H, sync), not a model"}
    return out


def run_ours(args, rank: int, local_rank: int, world: int):
    import gc
    import torch
    from paper_2606_08411_b200 import accounting, binding, workloads as W
    from paper_2606_08411_b200.step import HostStep

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()
    h = binding.Handle(local_rank)
    stream = torch.cuda.Stream(device=dev)
    sampler = ClockSampler(local_rank)
    sampler.start()

    wl = W.CONFIGS[args.workload]()
    acc = accounting.summary(wl)
    m = measure_resident(h, wl, dev, stream, dist, sampler, args.steps, args.warmup, args.kernel_events)
    step_ms, part_ms, launches_per_step = m["step_ms"], m["part_ms"], m["launches_per_step"]
    copies, n_copies, per_copy, barrier, first = m["copies"], m["n_copies"], m["per_copy"], m["barrier"], m["copies"][0]
    step_ms_max = max_over_ranks(step_ms, dist, dev)
    value = whole_job_value(acc["query_tokens"], world, step_ms_max)

    # ---- e2e: host buffers through al_lane_step_host (every layer of the workload, like `value`) --------
    hstep = HostStep(h, wl, device=dev)
    h2d, d2h = hstep.h2d_bytes, hstep.d2h_bytes
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    e2e_warm = min(3, args.warmup) or 1
    before = h.al_launch_count
    with torch.cuda.stream(stream):
        for i in range(e2e_warm):
            c = copies[i % n_copies]
            hstep.run(c.k_cache, c.v_cache, stream)
    e2e_launches = (h.al_launch_count - before) // e2e_warm
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.active.set()
    t0 = time.perf_counter()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in range(e2e_steps):
            c = copies[i % n_copies]
            hstep.run(c.k_cache, c.v_cache, stream)
        e1.record(stream)
    barrier()
    wall_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    sampler.active.clear()
    e2e_ms = max(e0.elapsed_time(e1) / e2e_steps, wall_ms)       # host-visible completion time
    e2e_ms = max_over_ranks(e2e_ms, dist, dev)
    e2e_tokens = wl.total_q_rows                                  # all layers of the workload per host step

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- the headline is measured FIRST, on a GPU that has done nothing yet (the fused LM head of `next_rows` draws
    # ~600 W and leaves this pool's B200s power-capped for a while); `clocks` is the sampler's view of the headline's
    # timed regions, `clocks_rest` that of everything measured afterwards
    clocks_headline = sampler.summary()
    sampler.reset()
    del hstep
    gc.collect()
    torch.cuda.empty_cache()
    # ---- then the other single-GPU configs (extra key `workloads`; fewer steps) and the 8(f) rows ----
    extra = {}
    if args.extra_workloads and world == 1:
        for name in [w for w in args.extra_workloads.split(",") if w and w != args.workload]:
            wl_x = W.CONFIGS[name]()
            acc_x = accounting.summary(wl_x)
            mx = measure_resident(h, wl_x, dev, stream, None, sampler, min(args.steps, args.extra_steps), args.warmup)
            parts_x = part_rooflines(wl_x, acc_x, mx["part_ms"], mx["step_ms"], peaks, load_traffic(wl_x.name))
            extra[wl_x.name] = {
                "step_us": mx["step_ms"] * 1e3, "query_tok_per_s": acc_x["query_tokens"] / (mx["step_ms"] * 1e-3),
                "steps": min(args.steps, args.extra_steps), "layers": wl_x.n_layers, "query_rows": wl_x.total_q_rows,
                "copies": mx["n_copies"], "gpu_launches_per_step": mx["launches_per_step"],
                "warm_l2_step_us": mx["warm_ms"] * 1e3 if mx["warm_ms"] else None,     # one copy replayed (fits the L2); step_us is the cold figure
                "parts": {k: {kk: p[kk] for kk in ("bound", "ms", "achieved", "peak", "unit", "frac", "traffic", "note") if kk in p}
                          for k, p in parts_x.items()}}
            del mx, wl_x
            gc.collect()
            torch.cuda.empty_cache()

    next_rows = None
    if args.next_rows and world == 1:
        next_rows = measure_next_rows(h, dev, stream, peaks)
        gc.collect()
        torch.cuda.empty_cache()

    clocks_rest = sampler.summary()
    sampler.stop_flag.set()
    sampler.join(timeout=2)

    # ---- roofline of every part; `roofline` = the part with the largest share of the step ------
    parts = {}
    if part_ms:
        parts = part_rooflines(wl, acc, part_ms, step_ms, peaks, load_traffic(wl.name))
        dom = max(parts, key=lambda k: parts[k]["ms"])
        roofline = {k: parts[dom][k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "note") if k in parts[dom]}
        roofline.update(kernel=dom, peak_source=peaks["source"], avg_launch_ms=parts[dom]["ms"] / parts[dom]["launches"],
                        timed_with="CUDA events on the stream around replays of a graph that runs the part on every resident copy in turn (consecutive launches share nothing through L2), right after the timed region")
    else:
        roofline = None

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu, _ = time_oracle(wl, steps=args.cpu_steps, warmup=1, budget_s=args.cpu_budget)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": step_ms_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": wl.dtype, "data": "synthetic",
        "config": {"workload": wl.name, "layers": wl.n_layers, "lanes": wl.n_lanes, "groups": wl.n_groups,
                   "query_rows": wl.total_q_rows, "heads": f"{wl.n_q_heads}q/{wl.n_kv_heads}kv", "head_dim": wl.head_dim,
                   "max_prefix": wl.max_prefix_len, "refresh_rows": int(wl.refresh_pos.size),
                   "logits": list(wl.logits.shape), "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": f"rotating {n_copies} resident copies of every streamed buffer "
                         f"({n_copies * per_copy / 1e6:.0f} MB > 2x 126 MB L2), one CUDA graph per step",
                   "graph": ("plan -> attention per layer -> {refresh on a side stream || confidence/select}"
                             if first.logits.numel() * first.logits.element_size() <= first.OVERLAP_MAX_LOGITS_BYTES
                             else "plan -> attention per layer -> refresh -> confidence/select")
                            + "; the parts are also timed alone on graphs of their own"},
        "clocks": clocks_headline, "clocks_rest": clocks_rest,
        "e2e": {"value": whole_job_value(e2e_tokens, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps, "layers": wl.n_layers,
                "api": "al_lane_step_host (pinned host buffers; H2D + plan + attention per layer + refresh + "
                       "confidence + D2H per step)",
                "gpu_launches_per_step": e2e_launches},
        "gpu_launches": launches_per_step * args.steps,
        "roofline": roofline, "parts": parts, "workloads": extra, "next_rows": next_rows, "cpu_baseline": cpu,
        "algorithmic": acc, "peaks": peaks,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)   # 71 ms at cfg5: past ~0.25 s of back-to-back steps this pool's B200s report sw_power_cap
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--extra-workloads", default="cfg2,cfg3,cfg4",
                    help="other configs measured in the same run and reported under `workloads` (N=1 only; '' = none)")
    ap.add_argument("--extra-steps", type=int, default=400)
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--cpu-steps", type=int, default=20)
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-events", dest="kernel_events", action="store_false")
    ap.add_argument("--no-next-rows", dest="next_rows", action="store_false",
                    help="skip the SURVEY 8(f) rows (fused LM head, lane status, refresh forward, scheduler) reported under `next_rows`")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
