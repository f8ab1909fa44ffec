"""CPU oracle of the AsyncLane host scheduler -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Algorithm 1 written out step by step in the paper's order, on top of the oracle's own
transfer rule (oracle.confidence_select, O-C) and lane status (oracle.lane_status, O-D).  It shares no code
with paper_2606_08411_b200/csrc/al_scheduler.cu; both follow the readings C18-C21 of DESIGN.md:

  * lane inputs (Eq.2): the lane's b tokens followed by a lookahead window of w = min(W, L - (s + b))
    rows for generate lanes (0 for refine lanes); prefix state kappa_l = cache rows [0, P + s) (L70)
  * transfer (L78-80): commit iff MASK and q >= tau; refine lanes suppress EOS; one token per lane is forced
    when nothing commits (finite denoising budget, reading C4)
  * fork (Eq.4-6): a generate lane forks when 0 < p < b, n_filled / b >= rho_min, t >= t_min and it
    still holds a MASK; refine child = [s, s + p) with a fresh clock, continuation = min(B, L - (s + p)) tokens
    from s + p
  * completion: no MASK left, or max_lane_steps updates; a completed, unforked generate lane spawns a successor
    at s + v unless v = 0 or s + v >= L (Eq.9, Alg.1 lines 10-17: cascading termination)
  * refresh (Eq.12) every refresh_period iterations: rows [0, min(P + L, P + L_eff + m)),
    L_eff = max over the tree of s + v
  * COLLECTDFS (L125): forked lanes emit their refine child, then their generate child; other lanes emit their
    own tokens up to the first MASK (generate lanes: or EOS), then their successor.

The stub model is part of the INPUT recipe (there are no weights): logits[row][v] = base[pos][v] + gain *
(step + 1) * (v == target[pos]) in float32, every term exactly representable.
"""
from __future__ import annotations

from typing import Dict, List

import numpy as np

from . import confidence_select, lane_status

GEN, REF = 0, 1
ACTIVE, COMPLETED, FORKED = 0, 1, 2


def stub_logits(base: np.ndarray, target: np.ndarray, gain: float, row_pos: np.ndarray, row_step: np.ndarray) -> np.ndarray:
    """float32 [n_rows][V]: base[pos] with gain * (step + 1) added at the position's target token."""
    x = base[row_pos].astype(np.float32).copy()
    x[np.arange(len(row_pos)), target[row_pos]] += np.float32(gain) * (row_step.astype(np.float32) + np.float32(1.0))
    return x


def run(cfg: Dict, base: np.ndarray, target: np.ndarray, gain: float, prompt: np.ndarray) -> Dict:
    P, L, B, W = cfg["prompt_len"], cfg["gen_len"], cfg["block_size"], cfg["lookahead"]
    mask, eos = cfg["mask_id"], cfg["eos_id"]
    tau, tau_f, rho = np.float32(cfg["tau"]), np.float32(cfg["tau_future"]), np.float32(cfg["rho_min"])
    delims, nofork = list(cfg["delimiter_ids"]), list(cfg["no_fork_prev_ids"])
    x = np.concatenate([np.asarray(prompt, np.int32), np.full(L, mask, np.int32)])
    nodes: List[Dict] = []

    def new_node(role, start, length, parent):
        nodes.append(dict(role=role, start=start, len=length, steps=0, parent=parent, ref_child=-1, gen_child=-1,
                          successor=-1, state=ACTIVE, valid_prefix=0, split_point=0, n_masked=length))
        return len(nodes) - 1

    new_node(GEN, 0, min(B, L), -1)
    stats = dict(iterations=0, model_calls=0, lane_forwards=0, forks=0, successors=0, refreshes=0, stopped_frontiers=0,
                 rows_forwarded=0, tokens_committed=0, tokens_drafted=0, refreshed_rows_last=0)
    refreshed = []                                   # L_refresh of every refresh, in order
    min_margin = 1.0                                 # how close any decided confidence came to a threshold
    while stats["iterations"] < cfg["max_iterations"]:
        active = [i for i, n in enumerate(nodes) if n["state"] == ACTIVE]
        if not active:
            break
        # ---- UPDATELANES (Alg.1 line 4): one batched model call for the active set ----
        lanes, toks, pos, step = [], [], [], []
        q_start = 0
        for i in active:
            n = nodes[i]
            s, b = n["start"], n["len"]
            w = min(W, L - (s + b)) if n["role"] == GEN else 0
            lanes.append([0, 0, P + s, q_start, b + w, (1 if n["role"] == REF else 0) | (w << 8)])
            toks.append(x[P + s:P + s + b + w]); pos.append(np.arange(s, s + b + w)); step.append(np.full(b + w, n["steps"]))
            q_start += b + w
        lanes = np.asarray(lanes, np.int32)
        toks, pos, step = np.concatenate(toks).astype(np.int32), np.concatenate(pos), np.concatenate(step)
        logits = stub_logits(base, target, gain, pos, step)
        sel = confidence_select(logits, toks, mask, eos, float(tau), lanes, force_top1=True)
        st = lane_status(lanes, toks, sel["conf"], sel["argmax"], mask, eos, float(tau_f), delims, nofork, sel["commit"],
                         sel["tokens_out"])
        masked_rows = toks == mask
        if masked_rows.any():
            min_margin = min(min_margin, float(np.abs(sel["conf"][masked_rows] - float(tau)).min()),
                             float(np.abs(sel["conf"][masked_rows] - float(tau_f)).min()))
        for k, i in enumerate(active):               # write back (L80) and advance the lane clocks
            n = nodes[i]
            qs, ql = int(lanes[k, 3]), int(lanes[k, 4])
            x[P + n["start"]:P + n["start"] + ql] = st["tokens_out"][qs:qs + ql]
            n["steps"] += 1
            n["valid_prefix"], n["split_point"], n["n_masked"] = (int(st["status"][k, 1]), int(st["status"][k, 2]),
                                                                 int(st["status"][k, 5]))
            n["n_filled"] = int(st["status"][k, 0])
            stats["tokens_committed"] += int(st["status"][k, 3]); stats["tokens_drafted"] += int(st["status"][k, 4])
        stats["model_calls"] += 1; stats["lane_forwards"] += len(active); stats["rows_forwarded"] += int(q_start)
        # ---- Alg.1 lines 5-17 ----
        for i in active:
            n = nodes[i]
            done = n["n_masked"] == 0 or n["steps"] >= cfg["max_lane_steps"]
            if n["role"] == REF:
                if done:
                    n["state"] = COMPLETED
                continue
            s, b, p, v = n["start"], n["len"], n["split_point"], n["valid_prefix"]
            fork = (0 < p < b and float(n["n_filled"]) >= float(rho) * b and n["steps"] >= cfg["t_min"] and n["n_masked"] > 0)
            if fork:                                  # Eq.6: F(l, p) = (l_ref, l_gen)
                n["ref_child"] = new_node(REF, s, p, i)
                n["gen_child"] = new_node(GEN, s + p, min(B, L - (s + p)), i)
                n["state"] = FORKED
                stats["forks"] += 1
            elif done:
                n["state"] = COMPLETED
                if v == 0 or s + v >= L:              # STOPADVANCE (Alg.1 line 13)
                    stats["stopped_frontiers"] += 1
                else:
                    n["successor"] = new_node(GEN, s + v, min(B, L - (s + v)), i)
                    stats["successors"] += 1
        stats["iterations"] += 1
        if cfg["refresh_period"] > 0 and stats["iterations"] % cfg["refresh_period"] == 0:
            l_eff = max(n["start"] + n["valid_prefix"] for n in nodes)
            l_refresh = min(P + L, P + l_eff + cfg["refresh_margin"])
            refreshed.append(l_refresh)
            stats["refreshes"] += 1; stats["refreshed_rows_last"] = l_refresh

    out: List[int] = []

    def emit(i):                                      # COLLECTDFS
        n = nodes[i]
        if n["state"] == FORKED:
            emit(n["ref_child"]); emit(n["gen_child"])
            return
        z = x[P + n["start"]:P + n["start"] + n["len"]]
        stop = (z == mask) | (z == eos) if n["role"] == GEN else (z == mask)
        cut = int(np.argmax(stop)) if stop.any() else len(z)
        out.extend(int(t) for t in z[:cut])
        if n["successor"] >= 0:
            emit(n["successor"])

    emit(0)
    for n in nodes:
        n.pop("n_filled", None)
    return dict(x=x, output=np.asarray(out, np.int32), tree=nodes, stats=stats, refreshed=refreshed,
                min_margin=min_margin)
