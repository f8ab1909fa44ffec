"""Seeded synthetic inputs for the lane-batched denoising step (data only).

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2606_08411_b200.binding``): it draws the inputs both sides consume.
It holds none of the method's arithmetic -- no attention, no softmax, no
confidence, no commit rule.  It only

* draws seeded Gaussian tensors and rounds them to the I/O dtype (so the rounded
  float32 values ARE the inputs of both sides),
* lays out lane / group descriptors (Eq.1) for the
  shapes BASELINE.json ``configs`` names,
* draws refresh positions (Eq.12) and token/mask states.

The paper gives no model shape and no hyper-parameter value; shapes come from
BASELINE.json ``configs`` (cfg1..cfg5 below = configs[0..4]).  The LLaDA/Dream
weights and the paper's benchmark datasets are not available, so these inputs
stand in for them ("Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

SEED_BASE = 20260608  # default_rng(20260608 + cfg_index)

# lane descriptor columns (int32), mirrors ``al_lane_desc`` in include/asynclane.h
LANE_GROUP_ID, LANE_KV_BASE_ROW, LANE_PREFIX_LEN, LANE_Q_START, LANE_Q_LEN, LANE_FLAGS = range(6)
LANE_FLAG_REFINE = 1


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 values to the nearest bfloat16 (ties to even); result stays float32."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def bf16_bits(x_rounded: np.ndarray) -> np.ndarray:
    """uint16 bit patterns of float32 values that are already bf16-representable."""
    return (np.ascontiguousarray(x_rounded, dtype=np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def _round(x: np.ndarray, dtype: str) -> np.ndarray:
    return round_to_bf16(x) if dtype == "bf16" else np.ascontiguousarray(x, dtype=np.float32)


def _normal(rng: np.random.Generator, shape, sigma: float, dtype: str) -> np.ndarray:
    x = rng.standard_normal(size=shape, dtype=np.float32)
    if sigma != 1.0:
        x *= np.float32(sigma)
    return _round(x, dtype)


@dataclass
class LaneStepWorkload:
    """One batch of inputs for one lane-batched denoising step.

    All floating tensors are float32 arrays whose values are exactly representable
    in ``dtype``.  Layouts follow include/asynclane.h.
    """

    name: str
    dtype: str                      # "f32" | "bf16"
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    n_layers: int
    cache_rows: int                 # capacity (rows) of one kv-head plane
    lanes: np.ndarray               # int32 [n_lanes, 6]
    q: np.ndarray                   # [L, T, H_q, d]
    k_new: np.ndarray               # [L, T, H_kv, d]
    v_new: np.ndarray               # [L, T, H_kv, d]
    k_cache: np.ndarray             # [L, H_kv, cache_rows, d]
    v_cache: np.ndarray             # [L, H_kv, cache_rows, d]
    refresh_pos: np.ndarray         # int32 [R] strictly increasing, relative to refresh_base_row
    refresh_base_row: int
    k_src: np.ndarray               # [L, R, H_kv, d]
    v_src: np.ndarray               # [L, R, H_kv, d]
    logits: np.ndarray              # [N, V]
    tokens: np.ndarray              # int32 [N]
    mask_id: int
    eos_id: int
    threshold: float
    planted_rows: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))
    notes: Dict[str, object] = field(default_factory=dict)

    @property
    def n_lanes(self) -> int:
        return int(self.lanes.shape[0])

    @property
    def total_q_rows(self) -> int:
        return int(self.q.shape[1])

    @property
    def max_prefix_len(self) -> int:
        return int(self.lanes[:, LANE_PREFIX_LEN].max()) if self.n_lanes else 0

    @property
    def vocab(self) -> int:
        return int(self.logits.shape[1])

    @property
    def n_groups(self) -> int:
        return int(np.unique(self.lanes[:, LANE_GROUP_ID]).size) if self.n_lanes else 0


def make_lanes(groups: List[dict]) -> np.ndarray:
    """Pack lane descriptors.  ``groups``: list of dicts with keys kv_base_row, prefix_len
    (int, or per-lane list), q_lens (list of lane lengths), refine (optional per-lane bools).
    Lanes are emitted group after group with dense, ascending ``q_start``."""
    rows = []
    q_start = 0
    for gid, g in enumerate(groups):
        q_lens = list(g["q_lens"])
        pl = g["prefix_len"]
        pls = list(pl) if isinstance(pl, (list, tuple, np.ndarray)) else [int(pl)] * len(q_lens)
        refine = list(g.get("refine", [False] * len(q_lens)))
        for j, ql in enumerate(q_lens):
            rows.append([gid, int(g["kv_base_row"]), int(pls[j]), q_start, int(ql),
                         LANE_FLAG_REFINE if refine[j] else 0])
            q_start += int(ql)
    return np.asarray(rows, dtype=np.int32).reshape(-1, 6)


def make_logits(rng: np.random.Generator, n_rows: int, vocab: int, sigma: float, dtype: str,
                planted_rows: np.ndarray, peak: float = 8.0) -> np.ndarray:
    """Gaussian logits (second parameter of N(0,.) read as the standard deviation) with
    ``planted_rows`` given one dominant entry: planted logit := (largest other logit of the
    row) + ``peak`` at a uniformly drawn index (SURVEY.md 8(c) reading C9), then rounded."""
    x = rng.standard_normal(size=(n_rows, vocab), dtype=np.float32)
    x *= np.float32(sigma)
    if len(planted_rows):
        idx = rng.integers(0, vocab, size=len(planted_rows))
        for r, j in zip(planted_rows, idx):
            row = x[r]
            row[j] = -np.inf
            row[j] = row.max() + np.float32(peak)
    return _round(x, dtype)


def make_tokens(rng: np.random.Generator, n_rows: int, vocab: int, mask_id: int,
                masked_frac: float = 0.5) -> np.ndarray:
    tok = rng.integers(0, vocab, size=n_rows).astype(np.int32)
    tok[tok == mask_id] = 0
    masked = rng.random(n_rows) < masked_frac
    tok[masked] = mask_id
    return tok


def build_workload(name: str, seed: int, dtype: str, n_q_heads: int, n_kv_heads: int, head_dim: int,
                   n_layers: int, cache_rows: int, groups: List[dict], n_refresh: int,
                   refresh_base_row: int, refresh_span: int, vocab: int, logit_sigma: float,
                   planted_frac: float, mask_id: int, eos_id: int, threshold: float,
                   n_planted: Optional[int] = None, logits_rows: Optional[int] = None,
                   contiguous_refresh: bool = False) -> LaneStepWorkload:
    """Generic seeded builder; every cfgN below and the ragged test cases go through it."""
    rng = np.random.default_rng(seed)
    lanes = make_lanes(groups)
    T = int(lanes[:, LANE_Q_LEN].sum()) if lanes.size else 0
    L, Hq, Hkv, d = n_layers, n_q_heads, n_kv_heads, head_dim
    q = _normal(rng, (L, T, Hq, d), 1.0, dtype)
    k_new = _normal(rng, (L, T, Hkv, d), 1.0, dtype)
    v_new = _normal(rng, (L, T, Hkv, d), 1.0, dtype)
    k_cache = _normal(rng, (L, Hkv, cache_rows, d), 1.0, dtype)
    v_cache = _normal(rng, (L, Hkv, cache_rows, d), 1.0, dtype)
    if contiguous_refresh:
        pos = np.arange(n_refresh, dtype=np.int32)
    else:
        pos = np.sort(rng.choice(refresh_span, size=n_refresh, replace=False)).astype(np.int32)
    k_src = _normal(rng, (L, n_refresh, Hkv, d), 1.0, dtype)
    v_src = _normal(rng, (L, n_refresh, Hkv, d), 1.0, dtype)
    N = T if logits_rows is None else logits_rows
    if n_planted is None:
        n_planted = int(round(planted_frac * N))
    planted = np.sort(rng.choice(N, size=n_planted, replace=False)) if n_planted else np.zeros(0, np.int64)
    logits = make_logits(rng, N, vocab, logit_sigma, dtype, planted)
    tokens = make_tokens(rng, N, vocab, mask_id)
    return LaneStepWorkload(name, dtype, Hq, Hkv, d, L, cache_rows, lanes, q, k_new, v_new,
                            k_cache, v_cache, pos, refresh_base_row, k_src, v_src, logits, tokens,
                            mask_id, eos_id, threshold, planted_rows=np.asarray(planted))


# ----------------------------------------------------------------------------------------------
# BASELINE.json configs[0..4]
# ----------------------------------------------------------------------------------------------

LLADA_VOCAB, LLADA_MASK_ID = 126464, 126336     # placeholders of the right size
DREAM_VOCAB, DREAM_MASK_ID = 152064, 151666


def cfg1_tiny() -> LaneStepWorkload:
    """configs[0]: tiny fp32 instance -- prefix 64, 2 lanes x 8, 2 heads MHA d=32, R=4,
    logits [16 x 512] ~ N(0, sigma=2) with 5 rows planted, threshold 0.9."""
    return build_workload("cfg1_tiny", SEED_BASE + 1, "f32", 2, 2, 32, 1, 96,
                          [dict(kv_base_row=0, prefix_len=64, q_lens=[8, 8], refine=[True, False])],
                          n_refresh=4, refresh_base_row=0, refresh_span=64,
                          vocab=512, logit_sigma=2.0, planted_frac=0.0, n_planted=5,
                          mask_id=511, eos_id=2, threshold=0.9)


def cfg2_llada_layer() -> LaneStepWorkload:
    """configs[1]: LLaDA-8B-shaped single layer bf16 -- 32 heads MHA d=128, prompt 256 +
    generated prefix 256, 4 lanes x 32 sharing it, R=32, logits [128 x 126464] ~ N(0, sigma=3),
    ~30% rows planted."""
    return build_workload("cfg2_llada_layer", SEED_BASE + 2, "bf16", 32, 32, 128, 1, 640,
                          [dict(kv_base_row=0, prefix_len=512, q_lens=[32] * 4,
                                refine=[True, False, True, False])],
                          n_refresh=32, refresh_base_row=0, refresh_span=512,
                          vocab=LLADA_VOCAB, logit_sigma=3.0, planted_frac=0.30,
                          mask_id=LLADA_MASK_ID, eos_id=126081, threshold=0.9)


def cfg3_dream_layer() -> LaneStepWorkload:
    """configs[2]: Dream-7B-shaped single layer bf16 -- GQA 28/4 d=128, prompt 512 + prefix 512,
    8 lanes x 32 in 2 fork groups (5+3) on distinct cache regions (reading C11), R=64,
    logits [256 x 152064] ~ N(0, sigma=3), 30% planted (stated choice)."""
    return build_workload("cfg3_dream_layer", SEED_BASE + 3, "bf16", 28, 4, 128, 1, 2304,
                          [dict(kv_base_row=0, prefix_len=1024, q_lens=[32] * 5,
                                refine=[True, False, True, False, False]),
                           dict(kv_base_row=1152, prefix_len=1024, q_lens=[32] * 3,
                                refine=[True, False, False])],
                          n_refresh=64, refresh_base_row=0, refresh_span=1024,
                          vocab=DREAM_VOCAB, logit_sigma=3.0, planted_frac=0.30,
                          mask_id=DREAM_MASK_ID, eos_id=151643, threshold=0.9)


def cfg4_long_llada(n_layers: int = 32) -> LaneStepWorkload:
    """configs[3]: long-generation LLaDA-shaped -- prompt 512 + gen 1024, lane tree depth 3,
    12 lanes x 32 in 4 groups at prefix lengths 512/768/1024/1280 (nested, one cache, reading
    C12), compact refresh of 320 rows (25% of 1280), 32 layers resident."""
    groups = [dict(kv_base_row=0, prefix_len=p, q_lens=[32] * 3, refine=[True, True, False])
              for p in (512, 768, 1024, 1280)]
    return build_workload("cfg4_long_llada", SEED_BASE + 4, "bf16", 32, 32, 128, n_layers, 1536,
                          groups, n_refresh=320, refresh_base_row=0, refresh_span=1280,
                          vocab=LLADA_VOCAB, logit_sigma=3.0, planted_frac=0.30,
                          mask_id=LLADA_MASK_ID, eos_id=126081, threshold=0.9)


def cfg5_lane_tree(rng: np.random.Generator, n_seqs: int, rows_per_seq: int) -> List[dict]:
    """Seeded random lane trees: per sequence prompt 384 + prefix U{384..768}, U{4..8} lanes x 32
    in 1..3 nested fork groups (deeper forks see a longer prefix of the same cache)."""
    groups = []
    for s in range(n_seqs):
        prefix_total = 384 + int(rng.integers(384, 769))
        n_lanes = int(rng.integers(4, 9))
        n_groups = int(rng.integers(1, 4))
        cuts = np.sort(rng.choice(np.arange(1, n_lanes), size=n_groups - 1, replace=False)) if n_groups > 1 else []
        sizes = np.diff(np.concatenate([[0], cuts, [n_lanes]])).astype(int)
        for j, sz in enumerate(sizes):
            plen = prefix_total - 64 * (n_groups - 1 - j)
            refine = [bool(rng.integers(0, 2)) for _ in range(sz)]
            refine[-1] = False
            groups.append(dict(kv_base_row=s * rows_per_seq, prefix_len=plen, q_lens=[32] * int(sz),
                               refine=refine))
    return groups


def cfg5_throughput_batch(n_seqs: int = 16) -> LaneStepWorkload:
    """configs[4]: throughput batch -- 16 independent Dream-shaped sequences (GQA 28/4, d=128),
    seeded random lane trees, logits over vocab 152064, 64 refreshed rows per sequence."""
    rows_per_seq = 1280
    rng = np.random.default_rng(SEED_BASE + 5)
    groups = cfg5_lane_tree(rng, n_seqs, rows_per_seq)
    wl = build_workload("cfg5_throughput_batch", SEED_BASE + 5, "bf16", 28, 4, 128, 1,
                        n_seqs * rows_per_seq, groups, n_refresh=0, refresh_base_row=0,
                        refresh_span=1, vocab=DREAM_VOCAB, logit_sigma=3.0, planted_frac=0.30,
                        mask_id=DREAM_MASK_ID, eos_id=151643, threshold=0.9)
    # 64 refreshed rows per sequence, as absolute (strictly increasing) pool rows
    pos = []
    for s in range(n_seqs):
        lo = s * rows_per_seq
        pos.append(lo + np.sort(rng.choice(768, size=64, replace=False)))
    wl.refresh_pos = np.concatenate(pos).astype(np.int32)
    R = wl.refresh_pos.size
    wl.k_src = _normal(rng, (1, R, 4, 128), 1.0, "bf16")
    wl.v_src = _normal(rng, (1, R, 4, 128), 1.0, "bf16")
    wl.notes["n_seqs"] = n_seqs
    return wl


def ragged_case(seed: int, dtype: str = "bf16", n_q_heads: int = 8, n_kv_heads: int = 2,
                head_dim: int = 128, n_groups: int = 3, vocab: int = 4099,
                max_prefix: int = 700) -> LaneStepWorkload:
    """Ragged-lane test case (not timed): lane lengths drawn from {11..24} U {32} after the fork
    position quartiles 11/17/24 of PAPER.md L266 Table 6; per-lane prefix lengths differ inside a
    group (reading C1); ragged vocab exercises the scalar head/tail of the confidence stream."""
    rng = np.random.default_rng(seed)
    groups = []
    base = 0
    for g in range(n_groups):
        n = int(rng.integers(1, 6))
        q_lens = [int(rng.choice(np.concatenate([np.arange(11, 25), [32]]))) for _ in range(n)]
        gp = int(rng.integers(1, max_prefix))
        pls = [max(0, gp - int(rng.integers(0, 40)) * int(rng.integers(0, 2))) for _ in range(n)]
        groups.append(dict(kv_base_row=base, prefix_len=pls, q_lens=q_lens,
                           refine=[bool(rng.integers(0, 2)) for _ in range(n)]))
        base += gp + int(rng.integers(0, 50))
    cache_rows = base + 160
    n_ref = int(rng.integers(1, 40))
    return build_workload(f"ragged_{seed}", seed, dtype, n_q_heads, n_kv_heads, head_dim, 1,
                          cache_rows, groups, n_refresh=n_ref, refresh_base_row=int(rng.integers(0, 16)),
                          refresh_span=cache_rows - 16, vocab=vocab, logit_sigma=3.0,
                          planted_frac=0.3, mask_id=vocab - 1, eos_id=int(rng.integers(0, vocab - 1)),
                          threshold=0.9)


CONFIGS = {
    "cfg1": cfg1_tiny,
    "cfg2": cfg2_llada_layer,
    "cfg3": cfg3_dream_layer,
    "cfg4": cfg4_long_llada,
    "cfg5": cfg5_throughput_batch,
}


def scheduler_case(seed: int, prompt_len: int = 24, gen_len: int = 160, block_size: int = 32, lookahead: int = 8,
                   vocab: int = 64, eos_frac: float = 0.8) -> Dict[str, object]:
    """Inputs of one scheduler run (Alg.1) with the table-driven stub model (there are no
    weights): a target "text" of sentences over token ids 20.., delimiter id 7 every 6..20 tokens (a third of
    them after the digit id 5: the numeric-period exclusion of L195), EOS (id 2) from eos_frac of the generation
    length on; `base` [gen_len][vocab] float32 logits in eighths (exactly representable), the target token's base
    logit in [-1, 3] so that positions reach the threshold after different numbers of steps while the target is
    the row maximum from the first step.  Data only: no arithmetic of the method."""
    rng = np.random.default_rng(seed)
    mask_id, eos_id, delim, digit = vocab - 1, 2, 7, 5
    target = rng.integers(20, vocab - 4, size=gen_len).astype(np.int32)
    i = int(rng.integers(6, 21))
    while i < gen_len:
        target[i] = delim
        if i > 0 and rng.random() < 0.33:
            target[i - 1] = digit
        i += int(rng.integers(6, 21))
    eos_at = int(eos_frac * gen_len)
    target[eos_at:] = eos_id                               # a finished sequence is padded with EOS
    base = (rng.integers(-24, -7, size=(gen_len, vocab)) / 8.0).astype(np.float32)        # others in [-3, -1]
    base[np.arange(gen_len), target] = (rng.integers(-8, 25, size=gen_len) / 8.0).astype(np.float32)   # [-1, 3]
    prompt = rng.integers(20, vocab - 4, size=prompt_len).astype(np.int32)
    cfg = dict(prompt_len=prompt_len, gen_len=gen_len, block_size=block_size, lookahead=lookahead, vocab=vocab,
               mask_id=mask_id, eos_id=eos_id, tau=0.9, tau_future=0.95, rho_min=0.5, t_min=2, max_lane_steps=24,
               max_iterations=400, refresh_period=4, refresh_margin=8, delimiter_ids=[delim], no_fork_prev_ids=[digit])
    return dict(cfg=cfg, base=base, target=target, gain=0.75, prompt=prompt, eos_at=eos_at)
