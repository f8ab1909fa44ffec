"""Host side of al_scheduler_run (Algorithm 1): packs a configuration, keeps the stub model's
tables and the optional device state resident, calls the C entry and unpacks the lane tree.  Marshalling only --
the control flow lives in csrc/al_scheduler.cu, the arithmetic in the kernels it calls."""
from __future__ import annotations

import ctypes
from typing import Dict, Optional

import numpy as np
import torch

from . import binding as B


def make_config(cfg: Dict, keep: list) -> B.al_sched_config:
    d = np.ascontiguousarray(cfg["delimiter_ids"], dtype=np.int32)
    n = np.ascontiguousarray(cfg["no_fork_prev_ids"], dtype=np.int32)
    keep += [d, n]                                     # the struct holds raw host pointers
    return B.al_sched_config(cfg["prompt_len"], cfg["gen_len"], cfg["block_size"], cfg["lookahead"], cfg["vocab"],
                             cfg["mask_id"], cfg["eos_id"], cfg["tau"], cfg["tau_future"], cfg["rho_min"], cfg["t_min"],
                             cfg["max_lane_steps"], cfg["max_iterations"], cfg["refresh_period"], cfg["refresh_margin"],
                             d.ctypes.data if d.size else None, int(d.size), n.ctypes.data if n.size else None, int(n.size))


def run_with_stub_model(handle: B.Handle, cfg: Dict, base: np.ndarray, target: np.ndarray, gain: float,
                        prompt: np.ndarray, device_state: Optional[B.al_sched_device_state] = None,
                        max_tree: int = 4096, device="cuda:0", model_fn=None, model_user=None) -> Dict:
    """Runs Algorithm 1 with the library's table-driven stub model (or `model_fn`, an AL_MODEL_FN)."""
    keep: list = []
    c = make_config(cfg, keep)
    dev = torch.device(device)
    base_d = torch.from_numpy(np.ascontiguousarray(base, dtype=np.float32)).to(dev)
    target_d = torch.from_numpy(np.ascontiguousarray(target, dtype=np.int32)).to(dev)
    stub = B.al_stub_model(base_d.data_ptr(), target_d.data_ptr(), float(gain), int(cfg["vocab"]))
    lib = B.load_library()
    if model_fn is None:
        model_fn, model_user = lib.al_stub_model_fn, ctypes.addressof(stub)
    P, L = cfg["prompt_len"], cfg["gen_len"]
    x = np.zeros(P + L, np.int32)
    out = np.zeros(L, np.int32)
    tree = (B.al_sched_lane * max_tree)()
    prompt = np.ascontiguousarray(prompt, dtype=np.int32)
    n_out, n_tree, stats = handle.al_scheduler_run(c, model_fn, model_user, device_state, prompt, x, out, tree)
    names = [f[0] for f in B.al_sched_lane._fields_]
    nodes = [{k: int(getattr(tree[i], k)) for k in names} for i in range(n_tree)]
    return dict(x=x, output=out[:n_out].copy(), tree=nodes,
                stats={f[0]: int(getattr(stats, f[0])) for f in B.al_sched_stats._fields_ if f[0] != "reserved"})
