// K1 lane_attention (bf16, head_dim 128) on the 5th-generation tensor cores -- al_lane_attention's
// main path (Eq.2-3: each lane attends to its prefix state kappa_l and to its
// own rows; L168-172 Eq.11: lanes of one shared-prefix group are evaluated in one batched call).
//
// Work decomposition (built ON DEVICE from the lane descriptors by lane_plan_kernel, so the call is
// graph-replayable with new lanes; the plan depends only on the descriptors and is reused by every
// layer of one scheduler iteration, see al_lane_plan):
//   run      = maximal sequence of lanes adjacent in the array, of one group, contiguous in q_start
//   sub-tile = up to tpt = floor(128 / n_rep) consecutive tokens of a run; with the n_rep q-heads of
//              a kv-head stacked under every token it is a 128-row M tile of the tensor core
//   tile     = two consecutive sub-tiles A, B of a run (B may be empty): they share every prefix
//              K/V tile, so each K/V tile staged in shared memory feeds 2 x (128x128x128) MMAs
//   keys     = [prefix key tiles of 64 cache rows] ++ [local key tiles of 64 K_new rows covering the
//              lanes that intersect the tile]; every row masks what its own lane may not see
//   item     = (tile, kv-head): n_key_tiles steps of the main loop
// The 64-key steps of all items go to the CTAs in one of three ways: one CTA per item ("whole items")
// when every item can have a CTA of its own and splitting would not pay (small calls of this kind launch
// no plan kernel at all: every CTA derives its record itself, self_plan_record); whole items DEALT to
// the CTAs, longest first, when there are more items than CTAs and that is cheaper ("item lists"); else
// n_ctas contiguous ranges of the flattened steps of equal cost ("stream-K": steps + kEpiCost per item
// finished), a boundary within one step of an item boundary snapping to it.  An item
// whose steps are spread over several CTAs leaves one normalised fp32 partial + LSE per CTA in the
// workspace; the CTA that finishes last (a ticket counter per (item, sub-tile)) merges them in a
// fixed order -- no combine launch, bit-identical results from call to call.
// All CTAs that share (group, kv-head) read the same K/V tiles: HBM sees them once, L2 serves the
// rest -- "the prefix is read once per lane group" (BASELINE north_star).
//
// Main kernel, persistent, 384 threads, warp-specialised, one CTA per SM:
//   warp 0      TMA producer: both Q sub-tiles once per piece, K tiles through a 4-stage ring
//   warp 3      TMA producer of the V tiles (their stages are freed much later than the K stages)
//   warps 1, 2  MMA issuer of stream A / B (warp-uniform, one elected lane): S_b = Q_b.K^T (SS form)
//               into the stream's S buffer as soon as the softmax holds the previous S in registers;
//               O_b += P_b.V with P_b read from one of the stream's two P buffers in TMEM (TS form)
//               and V MN-major in shared memory.  (In the instance for one whole item of one sub-tile
//               warp 1 issues every Q.K^T and warp 2 every P.V, each for both streams.)
//   warps 4-7   softmax of stream A (sub-tile A), one thread per stacked row
//   warps 8-11  softmax of stream B (sub-tile B; with one sub-tile per tile under a whole-item plan
//               the two streams take alternate key tiles of it and the epilogue merges them)
//               O is rescaled lazily (only when the running max grows by more than 2^8).  Epilogue
//               per stream: normalise, stage 128-byte half rows in shared memory, store coalesced
//               (bf16 output: one TMA tensor store per 64-column half of a full sub-tile; fp32
//               partial for a split item: bulk stores).
// TMEM (512 columns): S_A | S_B (64 fp32 columns each) | P_A[2] | P_B[2] (32 columns of packed bf16
// each) | O_A | O_B (128 fp32 columns each).
#include <cuda_bf16.h>

#include "al_internal.h"
#include "al_ptx.cuh"
#include "al_debug.cuh"

using namespace alptx;

namespace {

constexpr int kBM = 128;                   // stacked query rows per tile
constexpr int kBN = 64;                    // keys per key tile (step); 64 leaves TMEM room for P buffers of their own (measured faster than 128)
constexpr int kD = 128;                    // head_dim
constexpr int kStagesK = 256 / kBN;                // K ring depth (a K tile lives until its Q.K^T has run)
constexpr int kStagesV = 256 / kBN;                // V ring depth (a V tile lives until its P.V has run)
constexpr int kHalfBytes = kBM * 64 * 2;   // Q: [128 rows][64 bf16] = one 128-byte-swizzled half tile
constexpr int kKvHalfBytes = kBN * 64 * 2; // K, V: [64 keys][64 bf16]
constexpr int kTileBytes = 2 * kKvHalfBytes;
constexpr int kThreads = 384;             // warps 0-3: K loads, Q.K^T issue, P.V issue, V loads; 4-11: softmax of streams A, B
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: P <= 2^8 between rescales
constexpr int kMaxPlanLanes = 1024;
constexpr int kMaxPlanTiles = 2048;
constexpr int kPlanThreads = 256;
constexpr int kPlanTilesInSmem = 96;
constexpr int kMaxCtas = 256;              // >= SMs of any sm_100 part
constexpr int kMinPiece = 256 / kBN;       // do not cut the work finer than 256 keys per CTA
#ifndef AL_EPI_COST
#define AL_EPI_COST 4
#endif
constexpr int kEpiCost = AL_EPI_COST;      // what the epilogue of an item costs, in 64-key steps, when the step ranges are cut
constexpr int kPieceCost = 3;              // what a whole piece costs besides its steps (drain, epilogue, restart), in steps: measured 2.8 us
constexpr int kSplitPieceCost = 6;         // ... and a piece of a split item (fp32 partial, ticket, its share of the merge): measured 5.8 us
constexpr int kDealMaxTiles = 512;         // item-list plans rank the tiles by counting: n_tiles^2 / 256 smem reads per thread
constexpr int kSplitCost = 1280 / kBN;     // what splitting an item costs (partial epilogue, ticket, merge by the last CTA), in steps: measured 12-20 us

struct __align__(16) TileRec {             // 64 bytes
  int q_tok0, n_tok;          // first packed token row, tokens in the tile (<= 2 tpt)
  int kv_base_row;            // cache row of prefix key 0
  int kv_len_max, kv_len_min; // largest / smallest prefix_len among the lanes of the tile
  int lk0, lk1;               // local keys: packed rows [lk0, lk1) of K_new / V_new
  int lane_first, lane_count;
  int n_pref_tiles, n_key_tiles;
  int kt_off;                 // index of step (g = 0, kt = 0) of this tile in the flattened sequence
  int sub_lk0[2], sub_lk1[2]; // local key rows the lanes of sub-tile A / B can see (lk0 > lk1: none)
};
struct __align__(16) CtaRec {              // 112 bytes; the ONE record a CTA reads before it can issue its first loads
  int f_begin, f_end;         // this CTA's range of the flattened step sequence (item-list plans: of `order`)
  int tile0;                  // tile that contains f_begin
  int first_c0, first_c1;     // CTAs that hold pieces of the item this CTA's FIRST step belongs to
  int last_c0, last_c1;       // same for the item of its LAST step
  int pad;                    // item-list plans: id of the CTA's first item
  TileRec first;              // copy of tiles[tile0]: one load instead of two dependent ones at kernel start
  int flags;                  // kCtaActive | kCtaAlt | kCtaLists (copies of the plan header's switches)
  int reserved[3];
};
constexpr int kCtaActive = 1, kCtaAlt = 2, kCtaLists = 4;
static_assert(sizeof(CtaRec) == 112, "CtaRec is loaded as seven 16-byte vectors");
struct PlanHeader {
  int n_tiles, n_items, k_total, n_ctas;
  int alt;           // tiles of one sub-tile are worked on by both streams (chosen with the whole-item mode)
  int item_lists;    // 1: a CTA's [f_begin, f_end) indexes `order` (whole items dealt to the CTAs); 0: flattened steps
  int pad[2];
};

struct Plan {
  PlanHeader* hdr;
  TileRec* tiles;
  CtaRec* ctas;
  int* bounds;       // [n_ctas + 1]
  int* counters;     // [n_items][2] tickets per (item, sub-tile), zero between calls (the merging CTA resets its item's)
  int* order;        // [n_items] item-list plans: item ids (tile * n_kv + kv-head), CTA after CTA
  float* part_o;     // [2 * grid][256][128]  slot 2c: CTA c's first piece, 2c+1: its last piece
  float* part_lse;   // [2 * grid][256]          (rows 128.. belong to sub-tile B)
};

struct Bounds {
  int max_tiles, grid;
};

__host__ __device__ inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// ---------------------------------------------------------------------------------------------
// plan: lanes -> runs -> tiles -> flattened steps -> per-CTA ranges.  One CTA, every stage parallel.
// ---------------------------------------------------------------------------------------------
// In-place exclusive scan of a[0, n) by the whole block; returns the total.
__device__ int block_exclusive_scan(int* a, int n, int* s_warp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  int carry = 0;
  for (int base = 0; base < n; base += blockDim.x) {
    const int i = base + threadIdx.x;
    const int v = i < n ? a[i] : 0;
    int x = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, x, off);
      if (lane >= off) x += y;
    }
    if (lane == 31) s_warp[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int w = lane < n_warps ? s_warp[lane] : 0;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, w, off);
        if (lane >= off) w += y;
      }
      s_warp[lane] = w;
    }
    __syncthreads();
    const int incl = x + (warp ? s_warp[warp - 1] : 0);
    const int total = s_warp[n_warps - 1];
    if (i < n) a[i] = carry + incl - v;
    __syncthreads();
    carry += total;
  }
  return carry;
}
// largest i in [0, n) with a[i] <= x   (a ascending, a[0] <= x)
__device__ __forceinline__ int last_le(const int* a, int n, int x) {
  int lo = 0, hi = n - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (a[mid] <= x) lo = mid; else hi = mid - 1;
  }
  return lo;
}

__global__ void __launch_bounds__(kPlanThreads)
lane_plan_kernel(const al_lane_desc* __restrict__ lanes, int n_lanes, int n_kv_heads, int tpt, Bounds bounds,
                 Plan plan) {
  __shared__ int s_qs[kMaxPlanLanes], s_qe[kMaxPlanLanes], s_pl[kMaxPlanLanes], s_kb[kMaxPlanLanes];
  __shared__ TileRec s_tiles[kPlanTilesInSmem];   // the first tiles, so that small plans need no global read-back
  __shared__ int s_run_lane0[kMaxPlanLanes + 1];
  __shared__ int s_a[kMaxPlanTiles + 1];       // scan scratch: run flags, tiles per run, steps per tile
  __shared__ int s_run_tile_base[kMaxPlanLanes + 1];
  __shared__ int s_bounds[kMaxCtas + 1];
  __shared__ int s_warp[32];
  __shared__ int s_max_nk;                     // longest item, in steps
  __shared__ int s_sorted[kDealMaxTiles];      // item-list plans: tile of rank r (longest first)
  __shared__ int s_makespan;
  __shared__ int s_tiles2;                     // tiles of the launch if every tile takes two sub-tiles
  const int tid = threadIdx.x;
  // programmatic dependent launch: the attention kernel may start its prologue (barriers, TMEM) now; it
  // waits for this grid's completion before it reads the plan
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  TRACE_P(0);
  if (tid == 0) { s_max_nk = 0; s_tiles2 = 0; }

  // runs
  for (int i = tid; i < n_lanes; i += blockDim.x) {
    const al_lane_desc b = lanes[i];
    s_qs[i] = b.q_start; s_qe[i] = b.q_start + b.q_len; s_pl[i] = b.prefix_len; s_kb[i] = b.kv_base_row;
    int start = 1;
    if (i > 0) {
      const al_lane_desc a = lanes[i - 1];
      start = !(a.group_id == b.group_id && a.kv_base_row == b.kv_base_row && a.q_start + a.q_len == b.q_start);
    }
    s_a[i] = start;
  }
  __syncthreads();
  TRACE_P(1);
  const int n_runs = block_exclusive_scan(s_a, n_lanes, s_warp);
  TRACE_P(2);
  for (int i = tid; i < n_lanes; i += blockDim.x) {
    const bool start = (i + 1 < n_lanes ? s_a[i + 1] : n_runs) != s_a[i];
    if (start) s_run_lane0[s_a[i]] = i;
  }
  if (tid == 0) s_run_lane0[n_runs] = n_lanes;
  __syncthreads();
  // tiles per run: two sub-tiles of tpt tokens per tile (they share every prefix K/V tile staged in shared memory).
  // Few tiles (twice as many items would still leave every item a CTA of its own): ONE sub-tile per tile, so that
  // both softmax streams of a CTA work on the same sub-tile's key tiles alternately (alt mode) and an item takes
  // half as many steps -- latency, not L2 traffic, is what such a launch pays for (cfg3: 32 items on 148 SMs).
  for (int r = tid; r < n_runs; r += blockDim.x) {
    const int l0 = s_run_lane0[r], l1 = s_run_lane0[r + 1];
    atomicAdd(&s_tiles2, ceil_div(max(0, s_qe[l1 - 1] - s_qs[l0]), 2 * tpt));
  }
  __syncthreads();
  const int tile_tok = (s_tiles2 > 0 && 4 * s_tiles2 * n_kv_heads <= min(bounds.grid, kMaxCtas)) ? tpt : 2 * tpt;
  for (int r = tid; r < n_runs; r += blockDim.x) {
    const int l0 = s_run_lane0[r], l1 = s_run_lane0[r + 1];
    s_run_tile_base[r] = ceil_div(max(0, s_qe[l1 - 1] - s_qs[l0]), tile_tok);
  }
  __syncthreads();
  TRACE_P(3);
  int n_tiles = block_exclusive_scan(s_run_tile_base, n_runs, s_warp);
  TRACE_P(4);
  n_tiles = min(n_tiles, min(bounds.max_tiles, kMaxPlanTiles));   // cannot bind when the lanes are disjoint
  // tiles
  for (int t = tid; t < n_tiles; t += blockDim.x) {
    const int r = last_le(s_run_tile_base, n_runs, t);
    const int l0 = s_run_lane0[r], l1 = s_run_lane0[r + 1];
    TileRec T;
    T.q_tok0 = s_qs[l0] + (t - s_run_tile_base[r]) * tile_tok;
    T.n_tok = min(tile_tok, s_qe[l1 - 1] - T.q_tok0);
    T.kv_base_row = s_kb[l0];
    T.kv_len_max = 0; T.kv_len_min = 0x7fffffff; T.lk0 = 0x7fffffff; T.lk1 = 0;
    T.sub_lk0[0] = T.sub_lk0[1] = 0x7fffffff; T.sub_lk1[0] = T.sub_lk1[1] = 0;
    const int lf = l0 + last_le(s_qs + l0, l1 - l0, T.q_tok0);    // lane that holds the tile's first token
    int l = lf;
    for (; l < l1 && s_qs[l] < T.q_tok0 + T.n_tok; ++l) {
      T.kv_len_max = max(T.kv_len_max, s_pl[l]);
      T.kv_len_min = min(T.kv_len_min, s_pl[l]);
      T.lk0 = min(T.lk0, s_qs[l]);
      T.lk1 = max(T.lk1, s_qe[l]);
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const int t0 = T.q_tok0 + b * tpt, t1 = min(t0 + tpt, T.q_tok0 + T.n_tok);
        if (s_qs[l] < t1 && s_qe[l] > t0) { T.sub_lk0[b] = min(T.sub_lk0[b], s_qs[l]); T.sub_lk1[b] = max(T.sub_lk1[b], s_qe[l]); }
      }
    }
    T.lane_first = lf; T.lane_count = l - lf;
    T.n_pref_tiles = ceil_div(T.kv_len_max, kBN);
    T.n_key_tiles = T.n_pref_tiles + ceil_div(T.lk1 - T.lk0, kBN);
    T.kt_off = 0;
    plan.tiles[t] = T;
    if (t < kPlanTilesInSmem) s_tiles[t] = T;
    s_a[t] = T.n_key_tiles * n_kv_heads;
    atomicMax(&s_max_nk, T.n_key_tiles);
  }
  __syncthreads();
  TRACE_P(5);
  const int k_total = block_exclusive_scan(s_a, n_tiles, s_warp);
  TRACE_P(6);
  if (tid == 0) s_a[n_tiles] = k_total;
  for (int t = tid; t < n_tiles; t += blockDim.x) plan.tiles[t].kt_off = s_a[t];
  // per-CTA ranges of the flattened step sequence
  const int grid = min(bounds.grid, kMaxCtas);
  int n_ctas = max(1, min(grid, ceil_div(k_total, kMinPiece)));
  // When every item can have a CTA of its own, cutting items only pays if the longest item costs more
  // than the balanced share plus what a split costs (fp32 partials, tickets, merge).
  __syncthreads();
  // steps per item of tile t, for t < kMaxPlanLanes, in the (now free) tiles-per-run scratch: the loops below
  // would otherwise divide by n_kv_heads per element
  int* s_nk = s_run_tile_base;
  for (int t = tid; t < min(n_tiles, kMaxPlanLanes); t += blockDim.x) s_nk[t] = (s_a[t + 1] - s_a[t]) / n_kv_heads;
  const bool whole_items = n_tiles > 0 && n_tiles * n_kv_heads <= grid &&
                           s_max_nk <= ceil_div(k_total, n_ctas) + kSplitCost;
  __syncthreads();
  if (whole_items) n_ctas = n_tiles * n_kv_heads;
  // ---- more items than CTAs: whole items DEALT to the CTAs instead of step ranges, when that is cheaper ----
  // Cutting the flattened steps into equal ranges leaves (nearly) every CTA with two pieces of split items,
  // and a split piece is the most expensive thing a CTA does (fp32 partial, ticket, merge: measured 5.8 us
  // against 1 us per step and 2.8 us per whole piece).  Dealing the items, longest first, forwards and
  // backwards over the CTAs ("snake") gives every CTA whole items only; the CTAs then differ by at most about
  // one item, which is compared with the estimated cost of the ranges.
  TRACE_P(7);
  const int n_items_all = n_tiles * n_kv_heads;
  if (!whole_items && n_items_all > grid && n_tiles <= kDealMaxTiles) {
    if (tid == 0) s_makespan = 0;
    for (int t = tid; t < n_tiles; t += blockDim.x) {        // rank of tile t among the tiles, longest first
      const int nk = s_nk[t];
      int rank = 0;
      for (int u = 0; u < n_tiles; ++u) {
        const int nku = s_nk[u];
        rank += (nku > nk || (nku == nk && u < t)) ? 1 : 0;
      }
      s_sorted[rank] = t;
    }
    __syncthreads();
    TRACE_P(8);
    // item j of the sorted sequence = (tile s_sorted[j / n_kv], kv-head j % n_kv).  With R = items / CTAs and rem
    // items left over, the CTAs fall into two classes: the first C - rem take R items each out of the LONGEST
    // (C - rem) R items, the other rem take R + 1 out of the rest -- so that the CTAs with one item more get the
    // shorter ones -- and inside a class round k deals its items forwards (k even) or backwards (k odd) over the
    // class's CTAs ("snake").  (One snake over all CTAs gives the extra item of an even R to the CTAs that already
    // hold the longest: cfg5, 408 items of 13-19 steps on 148 CTAs: makespan 56 against 54.)
    const int C = grid, R = n_items_all / C, rem = n_items_all - R * C;
    const int nA = C - rem;                                  // CTAs with R items; they take sorted items [0, nA R)
    auto deal = [&](int c, int k) {                          // sorted index of the k-th item of CTA c
      const bool a = c < nA;
      const int n = a ? nA : rem, cc = a ? c : c - nA;
      return (a ? 0 : nA * R) + k * n + ((k & 1) ? n - 1 - cc : cc);
    };
    for (int c = tid; c < C; c += blockDim.x) {
      const int count = R + (c < nA ? 0 : 1);
      int load = 0;
      for (int k = 0; k < count; ++k) load += s_nk[s_sorted[deal(c, k) / n_kv_heads]] + kPieceCost;
      atomicMax(&s_makespan, load);
    }
    __syncthreads();
    TRACE_P(9);
    const int ranges = ceil_div(k_total + kPieceCost * n_items_all, n_ctas) + 2 * kSplitPieceCost - kPieceCost;
    if (s_makespan <= ranges) {
      for (int c = tid; c < C; c += blockDim.x) {
        const int count = R + (c < nA ? 0 : 1);
        const int start = c < nA ? c * R : nA * R + (c - nA) * (R + 1);
        for (int k = 0; k < count; ++k) {
          const int j = deal(c, k);
          plan.order[start + k] = s_sorted[j / n_kv_heads] * n_kv_heads + j % n_kv_heads;
        }
        const int j0 = deal(c, 0);
        CtaRec Cr;
        Cr.f_begin = start; Cr.f_end = start + count;
        Cr.tile0 = s_sorted[j0 / n_kv_heads];
        Cr.first_c0 = Cr.first_c1 = Cr.last_c0 = Cr.last_c1 = c;
        Cr.pad = Cr.tile0 * n_kv_heads + j0 % n_kv_heads;      // the CTA's first item
        Cr.flags = kCtaActive | kCtaLists; Cr.reserved[0] = Cr.reserved[1] = Cr.reserved[2] = 0;
        Cr.first = Cr.tile0 < kPlanTilesInSmem ? s_tiles[Cr.tile0] : plan.tiles[Cr.tile0];   // written by this block above
        plan.ctas[c] = Cr;
      }
      for (int i = tid; i < 2 * n_items_all; i += blockDim.x) plan.counters[i] = 0;
      if (tid == 0) {
        plan.hdr->n_tiles = n_tiles; plan.hdr->n_items = n_items_all;
        plan.hdr->k_total = k_total; plan.hdr->n_ctas = C;
        plan.hdr->alt = 0; plan.hdr->item_lists = 1;
      }
      TRACE_P(10);
      return;
    }
  }
  TRACE_P(11);
  if (whole_items) {                                     // CTA c = item c = (tile c / n_kv, head c % n_kv): no searches
    for (int c = tid; c <= n_ctas; c += blockDim.x) {
      const int t = c / n_kv_heads, g = c - t * n_kv_heads;
      const int f0 = c == n_ctas ? k_total : s_a[t] + g * s_nk[t];
      plan.bounds[c] = f0;
      if (c < n_ctas) {
        CtaRec C;
        C.f_begin = f0; C.f_end = f0 + s_nk[t];
        C.tile0 = t;
        C.first_c0 = C.first_c1 = C.last_c0 = C.last_c1 = c;
        C.pad = c;
        C.reserved[0] = C.reserved[1] = C.reserved[2] = 0;
        C.first = t < kPlanTilesInSmem ? s_tiles[t] : plan.tiles[t];   // written by this block above
        C.first.kt_off = s_a[t];
        // a whole item of ONE sub-tile is worked on by both streams (alt instance of the roles); one of two
        // sub-tiles runs in the other instance, a stream per sub-tile
        C.flags = kCtaActive | (C.first.n_tok <= tpt ? kCtaAlt : 0);
        plan.ctas[c] = C;
      }
    }
    for (int c = n_ctas + tid; c < grid; c += blockDim.x) plan.ctas[c].flags = kCtaAlt;   // idle CTAs
    for (int i = tid; i < 2 * n_items_all; i += blockDim.x) plan.counters[i] = 0;
    if (tid == 0) {
      plan.hdr->n_tiles = n_tiles; plan.hdr->n_items = n_items_all;
      plan.hdr->k_total = k_total; plan.hdr->n_ctas = k_total > 0 ? n_ctas : 0;
      // with one item per CTA a single-sub-tile item would leave half of the CTA's softmax threads idle: both
      // streams work on it, taking alternate key tiles
      plan.hdr->alt = 1; plan.hdr->item_lists = 0;
    }
    TRACE_P(12);
    return;
  }
  const bool snap = k_total / n_ctas >= 4;
  for (int c = tid; c <= n_ctas; c += blockDim.x) {
    int f = (int)((long long)c * k_total / n_ctas);
    if (whole_items) {                                 // CTA c = item c = (tile c / n_kv, head c % n_kv)
      const int t = c / n_kv_heads;
      f = c == n_ctas ? k_total : s_a[t] + (c - t * n_kv_heads) * ((s_a[t + 1] - s_a[t]) / n_kv_heads);
    } else if (kEpiCost > 0 && c > 0 && c < n_ctas) {
      // equal shares of (steps + kEpiCost per item): the CTA that finishes an item also pays its epilogue.
      // Tile t starts at cost s_a[t] + kEpiCost * n_kv * t; inside it every item costs nk + kEpiCost.
      const long long x = (long long)c * (k_total + (long long)kEpiCost * n_tiles * n_kv_heads) / n_ctas;
      int lo = 0, hi = n_tiles - 1;
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((long long)s_a[mid] + (long long)kEpiCost * n_kv_heads * mid <= x) lo = mid; else hi = mid - 1;
      }
      const int nk = (s_a[lo + 1] - s_a[lo]) / n_kv_heads;
      const int within = (int)(x - ((long long)s_a[lo] + (long long)kEpiCost * n_kv_heads * lo));
      const int g = within / (nk + kEpiCost), rem = within - g * (nk + kEpiCost);
      f = s_a[lo] + g * nk + min(rem, nk);
    }
    if (!whole_items && snap && c > 0 && c < n_ctas) {
      const int t = last_le(s_a, n_tiles, f);
      const int nk = (s_a[t + 1] - s_a[t]) / n_kv_heads;
      const int rem = (f - s_a[t]) % nk;           // steps into the item
      if (rem <= 1) f -= rem; else if (nk - rem <= 1) f += nk - rem;
    }
    s_bounds[c] = f;
  }
  __syncthreads();
  for (int c = tid; c <= n_ctas; c += blockDim.x) {
    plan.bounds[c] = s_bounds[c];
    if (c < n_ctas) {
      CtaRec C;
      C.f_begin = s_bounds[c]; C.f_end = s_bounds[c + 1];
      C.tile0 = n_tiles ? last_le(s_a, n_tiles, C.f_begin) : 0;
      C.first_c0 = C.first_c1 = C.last_c0 = C.last_c1 = c;
      C.pad = 0;
      C.flags = (n_tiles && s_bounds[c] < s_bounds[c + 1]) ? kCtaActive : 0;
      C.reserved[0] = C.reserved[1] = C.reserved[2] = 0;
      if (n_tiles) {
        C.first = C.tile0 < kPlanTilesInSmem ? s_tiles[C.tile0] : plan.tiles[C.tile0];   // written by this block above
        C.first.kt_off = s_a[C.tile0];
      }
      if (n_tiles && C.f_begin < C.f_end) {
        for (int e = 0; e < 2; ++e) {            // e = 0: item of the first step, 1: item of the last step
          const int f = e ? C.f_end - 1 : C.f_begin;
          const int t = last_le(s_a, n_tiles, f);
          const int nk = (s_a[t + 1] - s_a[t]) / n_kv_heads;
          const int f0 = s_a[t] + (f - s_a[t]) / nk * nk, f1 = f0 + nk;
          const int c0 = last_le(s_bounds, n_ctas + 1, f0);            // bounds[c0] <= f0 < bounds[c0 + 1]
          const int c1 = last_le(s_bounds, n_ctas + 1, f1 - 1);        // bounds[c1] <  f1 <= bounds[c1 + 1]
          if (e) { C.last_c0 = c0; C.last_c1 = c1; } else { C.first_c0 = c0; C.first_c1 = c1; }
        }
      }
      plan.ctas[c] = C;
    }
  }
  for (int c = n_ctas + tid; c < grid; c += blockDim.x) plan.ctas[c].flags = 0;            // idle CTAs
  for (int i = tid; i < 2 * n_tiles * n_kv_heads; i += blockDim.x) plan.counters[i] = 0;   // one per (item, sub-tile)
  if (tid == 0) {
    plan.hdr->n_tiles = n_tiles; plan.hdr->n_items = n_tiles * n_kv_heads;
    plan.hdr->k_total = k_total; plan.hdr->n_ctas = k_total > 0 ? n_ctas : 0;
    // with one item per CTA a single-sub-tile item would leave half of the CTA's softmax threads idle;
    // under stream-K the CTAs have long mixed ranges and the merge of the two streams does not pay
    plan.hdr->alt = whole_items ? 1 : 0;
    plan.hdr->item_lists = 0;
  }
  TRACE_P(12);
}

// ---------------------------------------------------------------------------------------------
// main kernel
// ---------------------------------------------------------------------------------------------
// Of every eight column pairs of a key tile, those whose exp2 runs on the FMA pipes instead of the MUFU.
// With two sub-tiles per step both streams' softmax warps load each SM sub-partition's MUFU and three
// of eight pay; when the streams take alternate key tiles (whole-item plans) one of eight is enough and
// the instruction count matters more (cfg4: 648 -> 617 us with one, cfg5: 88.6 -> 90.9 us).
#ifndef AL_POLY_TWO
#define AL_POLY_TWO 0x52
#endif
#ifndef AL_POLY_ALT
#define AL_POLY_ALT 0x10
#endif
constexpr int kPolyMaskTwoSubTiles = AL_POLY_TWO, kPolyMaskAlt = AL_POLY_ALT;
#ifdef AL_EPI_NO_TMA_STORE
constexpr bool kTmaStoreOk = false;        // debug knob: every bf16 sub-tile is copied out by its own warps
#else
constexpr bool kTmaStoreOk = true;
#endif
#ifdef AL_NO_VZERO
#define AL_VZERO_ON 0
#else
#define AL_VZERO_ON 1
#endif
constexpr int kStagePitch = 128;           // 128 data bytes per staged row; 16-byte chunk c of row r sits at chunk c ^ (r & 7)

struct AttnSmem {
  alignas(1024) uint8_t q[2][2][kHalfBytes];           // [sub-tile][64-column half]
  alignas(1024) uint8_t k[kStagesK][2][kKvHalfBytes];
  alignas(1024) uint8_t v[kStagesV][2][kKvHalfBytes];
  alignas(1024) uint8_t stage[2 * kBM * kStagePitch];  // epilogue staging: 128 bytes of (stream b, row r) at row b*128 + r (source of the bulk stores)
  uint32_t stage_off[2 * kBM];                         // ... and where they go: global offset in units of 128 bytes
  uint64_t q_full, q_empty;
  uint64_t k_full[kStagesK], k_empty[kStagesK], v_full[kStagesV], v_empty[kStagesV];
  uint64_t s_full[2], s_free[2];           // [stream]: S written by Q.K^T / S in the softmax threads' registers
  uint64_t p_full[2][2], pv_done[2][2];    // [stream][P buffer]: P written / the P.V that read it has completed
  uint64_t o_full[2], o_empty[2];          // per piece: accumulator complete / read out
  CtaRec cta;                              // this CTA's plan record
  uint32_t tmem_base;
  int ticket[2][3];
  int alt_has[2];                          // alt mode: did stream b have key tiles in this piece
};
static_assert(sizeof(AttnSmem) <= 232448, "AttnSmem exceeds the 227 KB opt-in shared memory of sm_100");

struct AttnParams {
  const al_lane_desc* lanes;
  Plan plan;
  __nv_bfloat16* out;
  float* lse;
  int n_q_heads, n_kv_heads, n_rep, tpt;
  uint32_t q_box_bytes;                    // bytes of ONE sub-tile's Q box (both halves)
  float scale_log2;
  int n_lanes;
};

// One CTA's walk over its work: pieces (tile, g, [kt_begin, kt_end)).  Step-range plans: the CTA's range
// [f, f_end) of the flattened step sequence, items in (tile, kv-head) order, the first and last piece possibly
// parts of split items.  Item-list plans: whole items order[f .. f_end), in the order they were dealt.
struct PieceWalk {
  const TileRec* tiles;
  const int* order;
  int n_kv;
  bool lists;
  int f, f_end, t, g, kt;
  TileRec T;
  int kt_begin, kt_end;                    // the current piece
  int first_c0, first_c1, last_c0, last_c1;
  // C: the CTA's own record (a copy in shared memory, loaded once in the kernel prologue)
  __device__ __forceinline__ PieceWalk(const Plan& plan, const CtaRec* C, int n_kv_heads, int cta)
      : tiles(plan.tiles), order(plan.order), n_kv(n_kv_heads) {
    f = f_end = t = g = kt = 0;
    lists = false;
    first_c0 = first_c1 = last_c0 = last_c1 = cta;
    if (C->flags & kCtaActive) {
      lists = (C->flags & kCtaLists) != 0;
      f = C->f_begin; f_end = C->f_end; t = C->tile0;
      first_c0 = C->first_c0; first_c1 = C->first_c1; last_c0 = C->last_c0; last_c1 = C->last_c1;
      if (f < f_end) {
        T = C->first;
        if (lists) {
          g = C->pad - t * n_kv;           // pad = id of the CTA's first item
          kt = -1;                         // the first item is already in (t, g, T)
        } else {
          const int off = f - T.kt_off;
          g = off / T.n_key_tiles;
          kt = off - g * T.n_key_tiles;
        }
      }
    }
  }
  // Advances to the next piece; false when the work is exhausted.  After a true return T, g,
  // kt_begin, kt_end describe the piece.
  __device__ __forceinline__ bool next() {
    if (f >= f_end) return false;
    if (lists) {
      if (kt >= 0) {
        const int item = order[f];
        const int tt = item / n_kv;
        g = item - tt * n_kv;
        if (tt != t) { t = tt; T = tiles[t]; }
      }
      kt_begin = 0; kt_end = kt = T.n_key_tiles;
      ++f;
      return true;
    }
    if (kt == T.n_key_tiles) {             // previous piece ended its item
      kt = 0;
      if (++g == n_kv) { g = 0; T = tiles[++t]; }
    }
    kt_begin = kt;
    kt_end = min(T.n_key_tiles, kt + (f_end - f));
    f += kt_end - kt_begin;
    kt = kt_end;
    return true;
  }
  __device__ __forceinline__ bool whole() const { return kt_begin == 0 && kt_end == T.n_key_tiles; }
  __device__ __forceinline__ int item() const { return t * n_kv + g; }
};

// Which steps of a piece does stream b work on?  Two sub-tiles: stream b = sub-tile b (prefix tiles:
// always; local tiles: only those that hold rows of the lanes the sub-tile's tokens belong to).  One
// sub-tile ("alt" mode): even key tiles go to stream 0, odd ones to stream 1, each with its own running
// max, row sum and accumulator; the epilogue merges the two.  Worked out once per piece, so that the
// per-step test is two compares on registers (step i of the piece = key tile kt_begin + i).
struct StreamSteps {
  int pref;                                // steps [0, pref) are prefix tiles the stream takes
  int lo, n_loc;                           // steps [lo, lo + n_loc) are local tiles it takes
  int par;                                 // alt mode: it takes the steps with (i & 1) == par; else -1
  __device__ __forceinline__ StreamSteps(const TileRec& T, int tpt, int b, int kt_begin, bool alt_ok) {
    pref = 0; lo = 0; n_loc = 0; par = -1;
    if (alt_ok) {                          // a tile of one sub-tile (the CTA's record says so: kCtaAlt): the two streams take alternate key tiles of it
      par = (kt_begin ^ b) & 1;
    } else if (b * tpt < T.n_tok) {
      const int s0 = b ? T.sub_lk0[1] : T.sub_lk0[0], s1 = b ? T.sub_lk1[1] : T.sub_lk1[0];
      pref = T.n_pref_tiles - kt_begin;
      if (s1 > s0) {                       // local tile j holds rows [lk0 + 64 j, +64): those that meet [s0, s1)
        const int j0 = (s0 - T.lk0) / kBN, j1 = (s1 - T.lk0 + kBN - 1) / kBN;
        lo = T.n_pref_tiles + j0 - kt_begin; n_loc = j1 - j0;
      }
    }
  }
  __device__ __forceinline__ bool takes(int i) const {
    if (par >= 0) return (i & 1) == par;
    return i < pref || (unsigned)(i - lo) < (unsigned)n_loc;
  }
};

__device__ __forceinline__ void tmem_ld32_f(uint32_t taddr, float* dst) {
  uint32_t r[32];
  tmem_ld32(taddr, r);
#pragma unroll
  for (int i = 0; i < 32; ++i) dst[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void bar_sync_both() { asm volatile("bar.sync 3, 256;" ::: "memory"); }
__device__ __forceinline__ void bar_sync_stream(int b) { asm volatile("bar.sync %0, 128;" ::"r"(1 + b) : "memory"); }
__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ float ex2(float x) {             // x <= 8 here (or -inf)
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// packed fp32x2 arithmetic (sm_100): halves the FFMA / FADD issue slots of the softmax
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t ffma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t fadd2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// 2^x for a pair on the FMA pipes (the MUFU does 16 ex2 per clock and SM -- exactly the rate at which
// the tensor core produces scores, so half of the exponentials are taken off it): x = n + f with
// n = rint(x), f in [-0.5, 0.5]; 2^f by a degree-3 polynomial (relative error 7.5e-5, far below the bf16
// rounding of P); 2^n by adding n to the exponent field.  x is clamped at -126 (masked scores are -inf).
__device__ __forceinline__ void exp2_poly_pair(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  unpack2(x2, x0, x1);
  x2 = pack2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
  const uint64_t t2 = fadd2(x2, pack2(12582912.f, 12582912.f));            // 1.5 * 2^23: n lands in the low mantissa bits
  const uint64_t f2 = ffma2(fadd2(t2, pack2(-12582912.f, -12582912.f)), pack2(-1.f, -1.f), x2);
  uint64_t q2 = ffma2(pack2(0.055171460f, 0.055171460f), f2, pack2(0.24261086f, 0.24261086f));
  q2 = ffma2(q2, f2, pack2(0.69326097f, 0.69326097f));
  q2 = ffma2(q2, f2, pack2(0.99992812f, 0.99992812f));
  float q0, q1, t0, t1;
  unpack2(q2, q0, q1);
  unpack2(t2, t0, t1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}

// global row (token-major [T][H_q][d]) of stacked row r of sub-tile b
__device__ __forceinline__ long long out_row(const AttnParams& p, const TileRec& T, int g, int b, int r) {
  const int tl = r / p.n_rep;
  return (long long)(T.q_tok0 + b * p.tpt + tl) * p.n_q_heads + g * p.n_rep + (r - tl * p.n_rep);
}
__device__ __forceinline__ int sub_rows(const AttnParams& p, const TileRec& T, int b) {
  return max(0, min(p.tpt, T.n_tok - b * p.tpt)) * p.n_rep;
}

// Merge of the partials of sub-tile b of one split item by the 128 threads of stream b in the CTA
// that finished last.  Pieces of an item live on consecutive CTAs c0..c1: slot 2*c0+1 (c0's last
// piece), then 2*c for the rest.  Warp w owns rows [32w, 32w+32) in passes of kRows rows; a lane holds
// one float4 column group.  Per pass the loads of kBatch pieces (kRows coalesced 512-byte rows each,
// plus the rows' LSE in the low lanes) are all issued before any is used -- 32 loads in flight per
// lane, one L2 round trip; further pieces are folded in with a running maximum.  The order of
// operations is fixed, so the result does not depend on which CTA happens to arrive last.
template <int kBatch, int kRows>
__device__ __forceinline__ void merge_rows(const AttnParams& p, const TileRec& T, int g, int b, int c0, int n_pieces,
                                           int tid128) {
  const int warp = tid128 >> 5, lane = tid128 & 31;
  const int n_rows = __shfl_sync(0xffffffffu, sub_rows(p, T, b), 0);
  for (int pass = 0; pass < 32 / kRows; ++pass) {
    const int row0 = warp * 32 + pass * kRows;
    if (row0 >= n_rows) break;
    const int my_row = row0 + (lane & (kRows - 1));
    const bool has_row = my_row < n_rows;
    float mx = -INFINITY, wsum = 0.f;              // running maximum of the LSEs and sum of weights of lane's row
    float4 acc[kRows];
#pragma unroll
    for (int k = 0; k < kRows; ++k) acc[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    TRACE_M(11 + 0);
    for (int j0 = 0; j0 < n_pieces; j0 += kBatch) {
      float4 v[kBatch][kRows];
      float ls[kBatch];
#pragma unroll
      for (int jj = 0; jj < kBatch; ++jj) {
        const int j = j0 + jj;
        const int slot = j == 0 ? 2 * c0 + 1 : 2 * (c0 + j);
        const bool pj = j < n_pieces;
        ls[jj] = (pj && has_row) ? __ldcg(p.plan.part_lse + ((long long)slot * 2 + b) * kBM + my_row) : -INFINITY;
        // a partial is stored as the four 16 KB staging rounds it was written from (see part_round_ptr):
        // columns [32 q, 32 q + 32) of row r at round q, byte r * 128 + ((chunk ^ (r & 7)) << 4)
        const uint8_t* src = reinterpret_cast<const uint8_t*>(p.plan.part_o + ((long long)slot * 2 + b) * kBM * kD) +
                             (lane >> 3) * (kBM * kStagePitch);
#pragma unroll
        for (int k = 0; k < kRows; ++k) {
          const int rr = row0 + k;
          v[jj][k] = (pj && rr < n_rows)
                         ? __ldcg(reinterpret_cast<const float4*>(src + rr * kStagePitch + (((lane & 7) ^ (rr & 7)) << 4)))
                         : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
      TRACE_M(12);
      float mx_new = mx;
#pragma unroll
      for (int jj = 0; jj < kBatch; ++jj) mx_new = fmaxf(mx_new, ls[jj]);
      const float resc = (mx == -INFINITY) ? 0.f : exp2f((mx - mx_new) * kLog2e);     // 1 when the maximum stands
      wsum *= resc;
      mx = mx_new;
      float wj[kBatch];
#pragma unroll
      for (int jj = 0; jj < kBatch; ++jj) {
        wj[jj] = (ls[jj] == -INFINITY) ? 0.f : exp2f((ls[jj] - mx) * kLog2e);   // 0: the row saw no key in this piece
        wsum += wj[jj];
      }
      if (j0 > 0) {                                  // (the accumulators are zero before the first batch)
#pragma unroll
        for (int k = 0; k < kRows; ++k) {
          const float rk = __shfl_sync(0xffffffffu, resc, k);
          acc[k].x *= rk; acc[k].y *= rk; acc[k].z *= rk; acc[k].w *= rk;
        }
      }
#pragma unroll
      for (int jj = 0; jj < kBatch; ++jj) {
        // a piece in which none of these rows saw a key may hold stale memory (a stream without key tiles
        // in a piece writes nothing): skip it; rows without data inside a written piece hold zeros
        if (!__any_sync(0xffffffffu, wj[jj] > 0.f)) continue;
#pragma unroll
        for (int k = 0; k < kRows; ++k) {
          const float wk = __shfl_sync(0xffffffffu, wj[jj], k);
          acc[k].x = fmaf(wk, v[jj][k].x, acc[k].x); acc[k].y = fmaf(wk, v[jj][k].y, acc[k].y);
          acc[k].z = fmaf(wk, v[jj][k].z, acc[k].z); acc[k].w = fmaf(wk, v[jj][k].w, acc[k].w);
        }
      }
    }
    TRACE_M(13);
    const float inv = wsum > 0.f ? 1.0f / wsum : 0.f;
    int tl = row0 / p.n_rep, hl = row0 - tl * p.n_rep;                 // token and head of row0, carried along
    long long orow = (long long)(T.q_tok0 + b * p.tpt + tl) * p.n_q_heads + g * p.n_rep + hl;
#pragma unroll
    for (int k = 0; k < kRows; ++k) {                // all the shuffles first: the stores then do not wait for one each
      const float ik = __shfl_sync(0xffffffffu, inv, k);
      acc[k].x *= ik; acc[k].y *= ik; acc[k].z *= ik; acc[k].w *= ik;
    }
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      if (row0 + k < n_rows) {
        uint2 pk;
        pk.x = pack_bf16x2(acc[k].x, acc[k].y);
        pk.y = pack_bf16x2(acc[k].z, acc[k].w);
        reinterpret_cast<uint2*>(p.out + orow * kD)[lane] = pk;
      }
      if (++hl == p.n_rep) { hl = 0; orow += p.n_q_heads - p.n_rep + 1; } else ++orow;
    }
    if (p.lse && has_row && lane < kRows) p.lse[out_row(p, T, g, b, my_row)] = mx + logf(wsum);
    TRACE_M(14);
  }
}
__device__ __forceinline__ void merge_item(const AttnParams& p, const TileRec& T, int g, int b, int c0, int c1,
                                           int tid128) {
  const int n_pieces = c1 - c0 + 1;
  if (n_pieces <= 2) merge_rows<2, 16>(p, T, g, b, c0, n_pieces, tid128);   // the usual case: an item cut once
  else merge_rows<4, 8>(p, T, g, b, c0, n_pieces, tid128);
}

// Epilogue staging.  A thread writes the 128 bytes of its own row as eight 16-byte chunks; chunk c
// of row r is stored at chunk position c ^ (r & 7), which makes both the row-per-thread writes and the
// chunk-per-lane reads of the copy loop conflict-free without padding.
__device__ __forceinline__ void stage_chunk(uint8_t* my_stage, int r, int c, uint4 v) {
  *reinterpret_cast<uint4*>(my_stage + ((c ^ (r & 7)) << 4)) = v;
}
// Copies the staged rows [0, n_rows) of a stream to global memory with coalesced 16-byte accesses:
// 8 lanes per row, four rows per warp instruction; a warp copies the 32 rows its own threads staged.
// stage_off holds each row's global offset in units of 128 bytes (written by the row's own thread,
// which knows its token and head), so the loop is address-arithmetic free.
__device__ __forceinline__ void copy_out_rows(const uint8_t* stage_b, const uint32_t* off_b, int n_rows, int tid128,
                                              uint8_t* base) {
  const int warp = tid128 >> 5, lane = tid128 & 31;
  const int chunk = lane & 7;
  const int r0 = warp * 32 + (lane >> 3);
  uint4 v[8];
  uint32_t off[8];
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const int r = r0 + it * 4;
    v[it] = *reinterpret_cast<const uint4*>(stage_b + r * kStagePitch + ((chunk ^ (r & 7)) << 4));
    off[it] = off_b[r];
  }
#pragma unroll
  for (int it = 0; it < 8; ++it)
    if (r0 + it * 4 < n_rows) *reinterpret_cast<uint4*>(base + (size_t)off[it] * 128 + chunk * 16) = v[it];
}

// fp32 partial of (slot, sub-tile): four rounds of 32 columns, each the 16 KB image of a stream's staging
// rows (128 rows x 128 bytes, 16-byte chunks swizzled as stage_chunk writes them), stored by ONE bulk copy.
__device__ __forceinline__ float* part_round_ptr(const AttnParams& p, int slot, int sub, int round) {
  return p.plan.part_o + ((long long)slot * 2 + sub) * kBM * kD + round * (kBM * kStagePitch / 4);
}
// One epilogue round of a stream through its 16 KB of staging rows and the async proxy: wait until the
// bulk store that last read the staging rows is done with them, stage this round's 128 bytes per row,
// make them visible to the async proxy and let thread 0 of the stream issue the store.
#define AL_STAGE_ROUND_BEGIN()                                                                                 \
  do {                                                                                                         \
    if (tid128 == 0) bulk_wait_read_all();                                                                     \
    bar_sync_stream(b);                                                                                        \
  } while (0)
#define AL_STAGE_ROUND_END(issue_stmt)                                                                         \
  do {                                                                                                         \
    fence_proxy_async_smem();                                                                                  \
    bar_sync_stream(b);                                                                                        \
    if (tid128 == 0) { issue_stmt; bulk_commit(); }                                                            \
  } while (0)

// The role code of the kernel, compiled twice: FOR the "alt" mode (kAltOk: the CTA holds one whole item of one
// sub-tile, worked on by both streams -- `alt` is a compile-time constant) and without it (everything else:
// step ranges, item lists, whole items of two sub-tiles).  The plan (or self_plan_record) chooses per CTA.
// Keeping each mode's code out of the other instance is worth a lot: the general instance got 8 us of 108 at
// cfg5 in round 1, and making the alt instance alt-ONLY (it used to test the tile at run time) took cfg4 from
// 616 to 585 us per 32 layers and the cfg3 kernel from 18.4 to 16.7 us.
// The piece loops run ONCE in the alt instance: an alt CTA holds one whole item, and saying so lets the compiler fold
// the per-piece ring / phase counters (cfg4 562 -> 555 us per 32 layers, cfg2 kernel 13.3 -> 12.3 us).  (Also telling
// it that the piece starts at key tile 0 took the gain at cfg4 back: 564 us.)
#define AL_FOR_PIECES(w) for (bool more_ = (w).next(); more_; more_ = kAltOk ? false : (w).next())
template <bool kAltOk>
__device__ __forceinline__ void attn_roles(AttnSmem& sm, const AttnParams& p, const CUtensorMap* pmap_q,
                                           const CUtensorMap* pmap_knew, const CUtensorMap* pmap_vnew,
                                           const CUtensorMap* pmap_kc, const CUtensorMap* pmap_vc,
                                           const CUtensorMap* pmap_out, uint32_t tmem, int warp, int lane) {
  const bool active = (sm.cta.flags & kCtaActive) != 0;
  constexpr bool alt_ok = kAltOk;
  if (threadIdx.x == 0) TRACE(1);

  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
    if (warp == 0 && lane == 0 && active) {
      // ===================== TMA producer of Q and the K tiles =====================
      uint32_t kv_it = 0, piece_it = 0;
      PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
      AL_FOR_PIECES(w) {
        const TileRec& T = w.T;
        const bool two = !kAltOk && T.n_tok > p.tpt;      // (an alt CTA's item has one sub-tile)
        auto issue_k = [&](int kt) {
          const int sk = kv_it % kStagesK;
          const bool pref = kt < T.n_pref_tiles;
          const int row = pref ? T.kv_base_row + kt * kBN : T.lk0 + (kt - T.n_pref_tiles) * kBN;
          const CUtensorMap* mk = pref ? pmap_kc : pmap_knew;
          const int c1 = pref ? row : w.g, c2 = pref ? w.g : row;   // cache [g][row][d]; new rows [row][g][d]
          mbar_wait_relaxed(&sm.k_empty[sk], ((kv_it / kStagesK) & 1) ^ 1);
          mbar_arrive_expect_tx(&sm.k_full[sk], kTileBytes);
          tma_load_3d(sm.k[sk][0], mk, &sm.k_full[sk], 0, c1, c2);
          tma_load_3d(sm.k[sk][1], mk, &sm.k_full[sk], 64, c1, c2);
          ++kv_it;
        };
        int kt = w.kt_begin;
        // Cold start: all CTAs fill their rings at the same moment (148 x 192 KB: several microseconds of HBM
        // bandwidth), so what the first Q.K^T needs goes out first -- key tile 0, then Q, then key tile 1 -- and the
        // rest of the ring (and the V ring, below) only once key tile 0 has landed.
        if (piece_it == 0) issue_k(kt++);
        mbar_wait_relaxed(&sm.q_empty, (piece_it & 1) ^ 1);
        mbar_arrive_expect_tx(&sm.q_full, two ? 2 * p.q_box_bytes : p.q_box_bytes);   // a box is tpt*n_rep (<= 128) rows per half
        for (int b = 0; b < (two ? 2 : 1); ++b) {
          tma_load_3d(sm.q[b][0], pmap_q, &sm.q_full, 0, w.g * p.n_rep, T.q_tok0 + b * p.tpt);
          tma_load_3d(sm.q[b][1], pmap_q, &sm.q_full, 64, w.g * p.n_rep, T.q_tok0 + b * p.tpt);
        }
        TRACE(2);
        for (; kt < w.kt_end; ++kt) {
          if (piece_it == 0 && kv_it == 2) mbar_wait_relaxed(&sm.k_full[0], 0);
          issue_k(kt);
        }
        ++piece_it;
      }
    } else if (warp == 3 && lane == 0 && active) {
      // ===================== TMA producer of the V tiles =====================
      // (its own thread: a V stage is freed by P.V, long after the K stage of the same step, and K loads
      // must not queue behind it)
      uint32_t kv_it = 0;
      PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
      AL_FOR_PIECES(w) {
        const TileRec& T = w.T;
        for (int kt = w.kt_begin; kt < w.kt_end; ++kt, ++kv_it) {
          const int sv = kv_it % kStagesV;
          const bool pref = kt < T.n_pref_tiles;
          const int row = pref ? T.kv_base_row + kt * kBN : T.lk0 + (kt - T.n_pref_tiles) * kBN;
          const CUtensorMap* mv = pref ? pmap_vc : pmap_vnew;
          const int c1 = pref ? row : w.g, c2 = pref ? w.g : row;
          if (kv_it == 0) mbar_wait_relaxed(&sm.k_full[0], 0);   // cold start: behind key tile 0 (see the K producer)
          mbar_wait_relaxed(&sm.v_empty[sv], ((kv_it / kStagesV) & 1) ^ 1);
          mbar_arrive_expect_tx(&sm.v_full[sv], kTileBytes);
          tma_load_3d(sm.v[sv][0], mv, &sm.v_full[sv], 0, c1, c2);
          tma_load_3d(sm.v[sv][1], mv, &sm.v_full[sv], 64, c1, c2);
        }
      }
    } else if (!kAltOk && (warp == 1 || warp == 2) && active) {
      // ===================== MMA issuers of the step-range / item-list instance: warp 1 for stream A, warp 2 for stream B =====================
      // Per stream: S has one 64-column TMEM buffer, P (bf16, 32 columns) has two of its own.  The
      // softmax hands S back as soon as it holds the tile in registers, so Q.K^T of the stream's next
      // key tile runs under the softmax of the current one and depends on no P.V:
      //   QK(0) | QK(1) PV(0) | QK(2) PV(1) | ...      QK(i) waits for "S(i-1) read", PV(i) for P(i)
      // Two issuing threads keep one stream's wait for its softmax from holding up the other stream's
      // MMAs; both arrive on the K/V/Q stage barriers (count 2).  The whole warp runs the loop (uniform
      // control flow keeps descriptors and addresses in uniform registers); one elected lane issues the
      // tcgen05 instructions.
      const bool leader = elect_one();
      const int b = warp - 1;
      const uint32_t ts = tmem + b * kBN, tp = tmem + 128 + b * 64, to = tmem + 256 + b * 128;
      const uint32_t idesc_qk = make_idesc_bf16(kBM, kBN, 0, 0);
      const uint32_t idesc_pv = make_idesc_bf16(kBM, kD, 0, 1);
      // every descriptor is a constant plus a small address offset: build the bases once
      const uint64_t dq_own0 = make_desc_sw128(smem_u32(sm.q[b][0]), 16, 1024);
      const uint64_t dq_own1 = make_desc_sw128(smem_u32(sm.q[b][1]), 16, 1024);
      const uint64_t dq_a0 = make_desc_sw128(smem_u32(sm.q[0][0]), 16, 1024);
      const uint64_t dq_a1 = make_desc_sw128(smem_u32(sm.q[0][1]), 16, 1024);
      const uint64_t dk = make_desc_sw128(smem_u32(sm.k[0][0]), 16, 1024);               // + stage * (16 KB >> 4) + half * (8 KB >> 4)
      const uint64_t dv = make_desc_sw128(smem_u32(sm.v[0][0]), kKvHalfBytes, 1024);     // + stage * (16 KB >> 4)
      uint32_t kv_it = 0, piece_it = 0;
      uint32_t c_qk = 0, c_pv = 0;             // key tiles of this stream whose Q.K^T / P.V has been issued (all pieces)
      uint32_t oe = 0;                         // pieces so far in which the stream had key tiles: o_empty phase
      PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
      AL_FOR_PIECES(w) {
        const int n = w.kt_end - w.kt_begin;
        const bool alt = alt_ok;     // one sub-tile: both streams work on Q of sub-tile A
        const StreamSteps mine(w.T, p.tpt, b, w.kt_begin, alt_ok);
        const uint64_t dq0 = alt ? dq_a0 : dq_own0, dq1 = alt ? dq_a1 : dq_own1;
        mbar_wait(&sm.q_full, piece_it & 1);
        tc_fence_after();
        if (b == 0 && leader) TRACE(3);
        int owed = -1;                         // step (of the piece) of the key tile whose P.V is owed
        bool first = true;
        // A step only one stream works on (alt mode: every step): its issuer arrives twice on the K/V
        // stage barriers, which expect one arrival from each issuer, and the other issuer skips the step.
        const bool solo = alt;
        // O_b (+)= P . V of the owed key tile
#define AL_ISSUE_PV()                                                                                          \
        do {                                                                                                   \
          const uint32_t it_ = kv_it + owed;                                                                   \
          const int sv_ = it_ % kStagesV;                                                                      \
          const uint32_t u_ = c_pv & 1;                                                                        \
          if (leader) TRACE_TILE(8 + b, it_);                                                                  \
          mbar_wait(&sm.p_full[b][u_], (c_pv >> 1) & 1);                                                       \
          if (leader) TRACE_TILE(10 + b, it_);                                                                 \
          mbar_wait(&sm.v_full[sv_], (it_ / kStagesV) & 1);                                                    \
          if (leader && b == 0) TRACE_TILE(14, it_);                                                           \
          /* O_b of the stream's previous piece has been read out.  Only pieces in which the stream had     */ \
          /* key tiles complete a phase of o_empty[b] (oe counts them), so neither side can run ahead.      */ \
          if (first && oe > 0) mbar_wait(&sm.o_empty[b], (oe - 1) & 1);                                        \
          tc_fence_after();                                                                                    \
          /* keys of this tile that any row may see, rounded up to the MMA K step */                           \
          const int kt_ = w.kt_begin + owed;                                                                   \
          const int valid_ = kt_ < w.T.n_pref_tiles ? min(kBN, w.T.kv_len_max - kt_ * kBN)                     \
                                                    : min(kBN, w.T.lk1 - w.T.lk0 - (kt_ - w.T.n_pref_tiles) * kBN); \
          const int ksteps_ = (valid_ + 15) >> 4;                                                              \
          const uint64_t dv_ = dv + (uint64_t)(sv_ * (kTileBytes >> 4));                                       \
          if (ksteps_ == kBN / 16) {                /* the usual case: no per-MMA predicates */                \
            _Pragma("unroll")                                                                                  \
            for (int k = 0; k < kBN / 16; ++k)                                                                 \
              if (leader) mma_ts(to, tp + u_ * 32 + k * 8, dv_ + (uint64_t)(k * 128), idesc_pv, (!first || k) ? 1u : 0u); \
          } else {                                                                                             \
            /* ragged tail: the key rows [valid_, 16 ksteps_) of the V tile are rows no lane may see (cache  */ \
            /* rows beyond the group's longest prefix: unwritten or recycled memory).  P is exactly 0 there, */ \
            /* but 0 x NaN/Inf would still poison every row of the tile, so they are zeroed in shared memory */ \
            /* before the MMA reads them (both issuers may do it: same zeros).                               */ \
            if (AL_VZERO_ON && (valid_ & 15)) {                                                                 \
              const int nz_ = ksteps_ * 16 - valid_;                 /* 1..15 key rows of 128 bytes per half */ \
              for (int j_ = lane; j_ < nz_ * 16; j_ += 32) {                                                   \
                const int row_ = valid_ + (j_ >> 4), hc_ = j_ & 15;  /* half = hc_ >> 3, 16-byte chunk hc_ & 7 */ \
                *reinterpret_cast<uint4*>(sm.v[sv_][hc_ >> 3] + row_ * 128 + (hc_ & 7) * 16) = make_uint4(0u, 0u, 0u, 0u); \
              }                                                                                                \
              fence_proxy_async_smem();                                                                        \
              __syncwarp();                                                                                    \
            }                                                                                                  \
            _Pragma("unroll")                                                                                  \
            for (int k = 0; k < kBN / 16; ++k)                                                                 \
              if (leader && k < ksteps_) mma_ts(to, tp + u_ * 32 + k * 8, dv_ + (uint64_t)(k * 128), idesc_pv, (!first || k) ? 1u : 0u); \
          }                                                                                                    \
          if (leader) {                                                                                        \
            mma_commit(&sm.v_empty[sv_]);                                                                      \
            if (solo) mma_commit(&sm.v_empty[sv_]);                                                            \
            mma_commit(&sm.pv_done[b][u_]);                                                                    \
          }                                                                                                    \
          if (leader) TRACE_TILE(3 + 4 * b, it_);                                                              \
          first = false; ++c_pv; owed = -1;                                                                    \
        } while (0)
        for (int i = 0; i < n; ++i) {
          const uint32_t it = kv_it + i;
          const int sk = it % kStagesK;
          if (!mine.takes(i)) {
            // With two sub-tiles (local key tiles of one sub-tile's lanes only -- few) the idle issuer pays
            // what it owes and hands the stages back itself, once they have landed, which keeps the two
            // issuers within a stage phase.
            if (!alt) {
              if (owed >= 0) AL_ISSUE_PV();
              mbar_wait(&sm.k_full[sk], (it / kStagesK) & 1);
              if (leader) mma_commit(&sm.k_empty[sk]);
              mbar_wait(&sm.v_full[it % kStagesV], (it / kStagesV) & 1);
              if (leader) mma_commit(&sm.v_empty[it % kStagesV]);
            }
            continue;
          }
          if (leader && b == 0) TRACE_TILE(12, it);
          mbar_wait(&sm.k_full[sk], (it / kStagesK) & 1);
          if (leader && b == 0) TRACE_TILE(13, it);
          // ---- S_b = Q_b . K^T of step i, once the softmax holds the stream's previous S in registers
          if (c_qk > 0) mbar_wait(&sm.s_free[b], (c_qk - 1) & 1);
          tc_fence_after();
          if (b == 0 && leader) TRACE(4);
          const uint64_t dk0 = dk + (uint64_t)(sk * (kTileBytes >> 4)), dk1 = dk0 + (uint64_t)(kKvHalfBytes >> 4);
#pragma unroll
          for (int k = 0; k < 4; ++k) if (leader) mma_ss(ts, dq0 + (uint64_t)(2 * k), dk0 + (uint64_t)(2 * k), idesc_qk, k ? 1u : 0u);
#pragma unroll
          for (int k = 0; k < 4; ++k) if (leader) mma_ss(ts, dq1 + (uint64_t)(2 * k), dk1 + (uint64_t)(2 * k), idesc_qk, 1u);
          if (leader) {
            mma_commit(&sm.s_full[b]);
            mma_commit(&sm.k_empty[sk]);
            if (solo) mma_commit(&sm.k_empty[sk]);
          }
          if (leader) TRACE_TILE(4 * b, it);
          ++c_qk;
          if (owed >= 0) AL_ISSUE_PV();                      // P.V of the stream's previous key tile, behind this Q.K^T
          owed = i;
        }
        if (leader) mma_commit(&sm.q_empty);                 // this issuer's Q.K^T of the piece are all issued
        if (owed >= 0) AL_ISSUE_PV();
        if (leader && !first) mma_commit(&sm.o_full[b]);     // the piece's accumulator is complete
#undef AL_ISSUE_PV
        if (b == 0 && leader) TRACE(5);
        kv_it += n;
        if (!first) ++oe;
        ++piece_it;
      }
    } else if (kAltOk && warp == 1 && active) {
      // ===================== whole-item instance: Q.K^T issuer (both streams) =====================
      // Per stream: S has one 64-column TMEM buffer, P (bf16, 32 columns) has two of its own.  The
      // softmax hands S back as soon as it holds the tile in registers, so Q.K^T of the stream's next
      // key tile runs under the softmax of the current one and depends on no P.V:
      //   QK(0) | QK(1) PV(0) | QK(2) PV(1) | ...      QK(i) waits for "S(i-1) read", PV(i) for P(i)
      // In this instance Q.K^T and P.V are issued by DIFFERENT warps (P.V: warp 2 below), each for both streams:
      // QK(i+1) goes out as soon as S(i) is in registers, whatever the P.V warp is waiting for.  A whole-item
      // tile of one sub-tile alternates its key tiles between the streams, so each issuing warp has ONE stream's
      // work per step and a serial chain half as long as a per-stream issuer's (four barrier waits, twelve
      // MMAs, five commits, descriptor moves into uniform registers: ~2000 cycles per step by the debug
      // stamps).  Measured, kernel alone on L2-resident inputs: cfg3 20.1 -> 18.5 us, cfg4 618 -> 606 us per 32
      // layers; the step-range / item-list instance, where both streams take every step and each of these warps
      // would carry two streams' work, keeps one issuer per stream (cfg5: 59.9 us against 61.8 us split).
      // (Four issuing warps do not fit: the register file is split over the four SM sub-partitions and a
      // sub-partition holds two softmax warps of 216 registers plus ONE warp of 72.)  The whole warp runs the
      // loop (uniform control flow keeps descriptors and addresses in uniform registers); one elected lane
      // issues the tcgen05 instructions.
      const bool leader = elect_one();
      const uint32_t idesc_qk = make_idesc_bf16(kBM, kBN, 0, 0);
      // every descriptor is a constant plus a small address offset: build the bases once
      const uint64_t dq_a0 = make_desc_sw128(smem_u32(sm.q[0][0]), 16, 1024);
      const uint64_t dq_a1 = make_desc_sw128(smem_u32(sm.q[0][1]), 16, 1024);
      const uint64_t dq_b0 = make_desc_sw128(smem_u32(sm.q[1][0]), 16, 1024);
      const uint64_t dq_b1 = make_desc_sw128(smem_u32(sm.q[1][1]), 16, 1024);
      const uint64_t dk = make_desc_sw128(smem_u32(sm.k[0][0]), 16, 1024);               // + stage * (16 KB >> 4) + half * (8 KB >> 4)
      uint32_t kv_it = 0, piece_it = 0;
      uint32_t c_qk0 = 0, c_qk1 = 0;           // key tiles of stream A / B whose Q.K^T has been issued (all pieces)
      PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
      AL_FOR_PIECES(w) {
        const int n = w.kt_end - w.kt_begin;
        const bool alt = alt_ok;     // one sub-tile: both streams work on Q of sub-tile A
        const StreamSteps mine0(w.T, p.tpt, 0, w.kt_begin, alt_ok), mine1(w.T, p.tpt, 1, w.kt_begin, alt_ok);
        const uint64_t dq10 = alt ? dq_a0 : dq_b0, dq11 = alt ? dq_a1 : dq_b1;
        mbar_wait(&sm.q_full, piece_it & 1);
        tc_fence_after();
        if (leader) TRACE(3);
        for (int i = 0; i < n; ++i) {
          const uint32_t it = kv_it + i;
          const int sk = it % kStagesK;
          if (leader) TRACE_TILE(12, it);
          mbar_wait(&sm.k_full[sk], (it / kStagesK) & 1);
          if (leader) TRACE_TILE(13, it);
          const uint64_t dk0 = dk + (uint64_t)(sk * (kTileBytes >> 4)), dk1 = dk0 + (uint64_t)(kKvHalfBytes >> 4);
          // ---- S_b = Q_b . K^T of step i, once the softmax holds the stream's previous S in registers
#define AL_ISSUE_QK(b_, ts_, dq0_, dq1_, c_qk_)                                                                \
          do {                                                                                                 \
            if (c_qk_ > 0) mbar_wait(&sm.s_free[b_], (c_qk_ - 1) & 1);                                         \
            tc_fence_after();                                                                                  \
            if (b_ == 0 && leader) TRACE(4);                                                                   \
            _Pragma("unroll")                                                                                  \
            for (int k = 0; k < 4; ++k) if (leader) mma_ss(ts_, dq0_ + (uint64_t)(2 * k), dk0 + (uint64_t)(2 * k), idesc_qk, k ? 1u : 0u); \
            _Pragma("unroll")                                                                                  \
            for (int k = 0; k < 4; ++k) if (leader) mma_ss(ts_, dq1_ + (uint64_t)(2 * k), dk1 + (uint64_t)(2 * k), idesc_qk, 1u); \
            if (leader) mma_commit(&sm.s_full[b_]);                                                            \
            if (leader) TRACE_TILE(4 * b_, it);                                                                \
            ++c_qk_;                                                                                           \
          } while (0)
          if (mine0.takes(i)) AL_ISSUE_QK(0, tmem, dq_a0, dq_a1, c_qk0);
          if (mine1.takes(i)) AL_ISSUE_QK(1, tmem + kBN, dq10, dq11, c_qk1);
#undef AL_ISSUE_QK
          // the stage goes back when every Q.K^T issued so far has run (the barrier expects two arrivals)
          if (leader) { mma_commit(&sm.k_empty[sk]); mma_commit(&sm.k_empty[sk]); }
        }
        if (leader) { mma_commit(&sm.q_empty); mma_commit(&sm.q_empty); }   // the Q.K^T of the piece are all issued (the barrier expects two arrivals)
        if (leader) TRACE(5);
        kv_it += n;
        ++piece_it;
      }
    } else if (kAltOk && warp == 2 && active) {
      // ===================== whole-item instance: P.V issuer (both streams) =====================
      // O_b (+)= P . V of every key tile stream b takes, as soon as its softmax has stored P.
      const bool leader = elect_one();
      const uint32_t idesc_pv = make_idesc_bf16(kBM, kD, 0, 1);
      const uint64_t dv = make_desc_sw128(smem_u32(sm.v[0][0]), kKvHalfBytes, 1024);     // + stage * (16 KB >> 4)
      uint32_t kv_it = 0;
      uint32_t c_pv0 = 0, c_pv1 = 0;           // key tiles of stream A / B whose P.V has been issued (all pieces)
      uint32_t oe0 = 0, oe1 = 0;               // pieces so far in which the stream had key tiles: o_empty phase
      PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
      AL_FOR_PIECES(w) {
        const int n = w.kt_end - w.kt_begin;
        const StreamSteps mine0(w.T, p.tpt, 0, w.kt_begin, alt_ok), mine1(w.T, p.tpt, 1, w.kt_begin, alt_ok);
        bool first0 = true, first1 = true;
        // the last step each stream takes: its accumulator is complete behind that P.V
        int last0 = -1, last1 = -1;
        for (int i = n - 1; i >= 0 && (last0 < 0 || last1 < 0); --i) {
          if (last0 < 0 && mine0.takes(i)) last0 = i;
          if (last1 < 0 && mine1.takes(i)) last1 = i;
        }
        for (int i = 0; i < n; ++i) {
          const uint32_t it_ = kv_it + i;
          const int sv_ = it_ % kStagesV;
          const uint64_t dv_ = dv + (uint64_t)(sv_ * (kTileBytes >> 4));
          // keys of this tile that any row may see, rounded up to the MMA K step
          const int kt_ = w.kt_begin + i;
          const int valid_ = kt_ < w.T.n_pref_tiles ? min(kBN, w.T.kv_len_max - kt_ * kBN)
                                                    : min(kBN, w.T.lk1 - w.T.lk0 - (kt_ - w.T.n_pref_tiles) * kBN);
          const int ksteps_ = (valid_ + 15) >> 4;
          bool v_ready = false;
#define AL_ISSUE_PV(b_, tp_, to_, c_pv_, oe_, first_, last_)                                                   \
          do {                                                                                                 \
            const uint32_t u_ = c_pv_ & 1;                                                                     \
            if (leader) TRACE_TILE(8 + b_, it_);                                                               \
            mbar_wait(&sm.p_full[b_][u_], (c_pv_ >> 1) & 1);                                                   \
            if (leader) TRACE_TILE(10 + b_, it_);                                                              \
            if (!v_ready) {                                                                                    \
              mbar_wait(&sm.v_full[sv_], (it_ / kStagesV) & 1);                                                \
              v_ready = true;                                                                                  \
              /* ragged tail: the key rows [valid_, 16 ksteps_) of the V tile are rows no lane may see (cache */ \
              /* rows beyond the group's longest prefix: unwritten or recycled memory).  P is exactly 0      */ \
              /* there, but 0 x NaN/Inf would still poison every row of the tile, so they are zeroed in      */ \
              /* shared memory before the MMA reads them.                                                    */ \
              if (AL_VZERO_ON && (valid_ & 15)) {                                                               \
                const int nz_ = ksteps_ * 16 - valid_;               /* 1..15 key rows of 128 bytes per half */ \
                for (int j_ = lane; j_ < nz_ * 16; j_ += 32) {                                                 \
                  const int row_ = valid_ + (j_ >> 4), hc_ = j_ & 15; /* half = hc_ >> 3, 16-byte chunk hc_ & 7 */ \
                  *reinterpret_cast<uint4*>(sm.v[sv_][hc_ >> 3] + row_ * 128 + (hc_ & 7) * 16) = make_uint4(0u, 0u, 0u, 0u); \
                }                                                                                              \
                fence_proxy_async_smem();                                                                      \
                __syncwarp();                                                                                  \
              }                                                                                                \
            }                                                                                                  \
            if (leader && b_ == 0) TRACE_TILE(14, it_);                                                        \
            /* O_b of the stream's previous piece has been read out.  Only pieces in which the stream had   */ \
            /* key tiles complete a phase of o_empty[b] (oe counts them), so neither side can run ahead.    */ \
            if (first_ && oe_ > 0) mbar_wait(&sm.o_empty[b_], (oe_ - 1) & 1);                                  \
            tc_fence_after();                                                                                  \
            if (ksteps_ == kBN / 16) {              /* the usual case: no per-MMA predicates */                \
              _Pragma("unroll")                                                                                \
              for (int k = 0; k < kBN / 16; ++k)                                                               \
                if (leader) mma_ts(to_, tp_ + u_ * 32 + k * 8, dv_ + (uint64_t)(k * 128), idesc_pv, (!first_ || k) ? 1u : 0u); \
            } else {                                                                                           \
              _Pragma("unroll")                                                                                \
              for (int k = 0; k < kBN / 16; ++k)                                                               \
                if (leader && k < ksteps_) mma_ts(to_, tp_ + u_ * 32 + k * 8, dv_ + (uint64_t)(k * 128), idesc_pv, (!first_ || k) ? 1u : 0u); \
            }                                                                                                  \
            if (leader) mma_commit(&sm.pv_done[b_][u_]);                                                       \
            if (leader && i == last_) mma_commit(&sm.o_full[b_]);    /* the piece's accumulator is complete */ \
            if (leader) TRACE_TILE(3 + 4 * b_, it_);                                                           \
            first_ = false; ++c_pv_;                                                                           \
          } while (0)
          if (mine0.takes(i)) AL_ISSUE_PV(0, tmem + 128, tmem + 256, c_pv0, oe0, first0, last0);
          if (mine1.takes(i)) AL_ISSUE_PV(1, tmem + 128 + 64, tmem + 256 + 128, c_pv1, oe1, first1, last1);
#undef AL_ISSUE_PV
          // the stage goes back when every P.V issued so far has run (two arrivals expected); a step neither
          // stream takes is handed back once it has landed
          if (!v_ready) mbar_wait(&sm.v_full[sv_], (it_ / kStagesV) & 1);
          if (leader) { mma_commit(&sm.v_empty[sv_]); mma_commit(&sm.v_empty[sv_]); }
        }
        kv_it += n;
        if (!first0) ++oe0;
        if (!first1) ++oe1;
      }
    }
  } else {
    // ===================== softmax + epilogue: stream b = sub-tile b, one thread per stacked row =====================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    const int b = (warp - 4) >> 2;                     // stream / sub-tile
    const int quad = warp & 3;                         // TMEM lane group this warp may access
    const int r = quad * 32 + lane;                    // row of the sub-tile
    const int tid128 = (threadIdx.x - 128) & 127;
    const uint32_t lane_addr = (uint32_t)(quad * 32) << 16;
    const uint32_t t_o = tmem + 256 + b * 128;
    const uint64_t scale2 = pack2(p.scale_log2, p.scale_log2);
    uint8_t* stage_b = sm.stage + b * kBM * kStagePitch;
    uint8_t* my_stage = stage_b + r * kStagePitch;
    uint32_t* off_b = sm.stage_off + b * kBM;
    uint32_t cnt = 0;                                  // key tiles this stream has processed (all pieces)
    uint32_t pieces_done = 0;                          // pieces in which it had key tiles: o_full phase
    PieceWalk w(p.plan, &sm.cta, p.n_kv_heads, blockIdx.x);
    AL_FOR_PIECES(w) {
      const TileRec& T = w.T;
      const int n = w.kt_end - w.kt_begin;
      const bool alt = alt_ok;     // one sub-tile: this stream takes every other key tile of it
      const int sb = alt ? 0 : b;                      // sub-tile whose rows this stream holds
      const StreamSteps mine(T, p.tpt, b, w.kt_begin, alt_ok);
      const int n_rows = sub_rows(p, T, sb);
      // ---- this row's token and lane ----
      const int tok_local = r / p.n_rep;
      const int tok = T.q_tok0 + sb * p.tpt + tok_local;
      bool valid = r < n_rows;
      int prefix_len = 0, ls = 0, le = 0;
      if (valid) {
        valid = false;
        for (int l = T.lane_first; l < T.lane_first + T.lane_count; ++l) {
          const int qs = p.lanes[l].q_start, ql = p.lanes[l].q_len;
          if (tok >= qs && tok < qs + ql) { prefix_len = p.lanes[l].prefix_len; ls = qs; le = qs + ql; valid = true; }
        }
      }
      float m_used = -INFINITY, l_sum = 0.f;           // m_used in raw score units
      int n_mine = 0;

      for (int i = 0; i < n; ++i) {
        const int kt = w.kt_begin + i;
        if (!mine.takes(i)) continue;
        const uint32_t u = cnt & 1;                      // P buffer of this key tile
        const uint32_t t_s = tmem + b * kBN, t_p = tmem + 128 + b * 64 + u * 32;
        TRACE_W(5);
        mbar_wait(&sm.s_full[b], cnt & 1);
        tc_fence_after();
        TRACE_W(6);
        if (tid128 == 0 && b == 0) TRACE(6);
        if (tid128 == 0) TRACE_TILE(1 + 4 * b, cnt);
        TRACE_W(0);
        float s[kBN];
#pragma unroll
        for (int c = 0; c < kBN / 32; ++c) tmem_ld32_f(t_s + lane_addr + c * 32, s + c * 32);
        tmem_wait_ld();
        tc_fence_before();
        mbar_arrive(&sm.s_free[b]);                      // S is in registers: the stream's next Q.K^T may overwrite it
        TRACE_W(1);
        // visible columns of this tile for this row: [lo, hi).  Rows beyond the sub-tile's last token are
        // never stored: they run unmasked on whatever their Q row holds.
        int lo = 0, hi = kBN;
        if (kt < T.n_pref_tiles) {
          hi = min(kBN, prefix_len - kt * kBN);
        } else {
          const int base = T.lk0 + (kt - T.n_pref_tiles) * kBN;
          lo = max(0, ls - base); hi = min(kBN, le - base);
        }
        const bool need_mask = valid && (lo > 0 || hi < kBN);
        uint32_t hidden = 0;                             // bit c: 32-column chunk c is entirely hidden from this row
        if (__any_sync(0xffffffffu, need_mask)) {        // warp-uniform: only ragged prefix tails and local tiles
          uint32_t vis[kBN / 32];                        // bit e of vis[c]: column 32 c + e is visible
#pragma unroll
          for (int c4 = 0; c4 < kBN / 32; ++c4) {
            const int a = min(32, max(0, lo - c4 * 32)), z = min(32, max(0, hi - c4 * 32));   // visible [a, z) of the chunk
            const uint32_t below_z = z >= 32 ? 0xffffffffu : ((1u << z) - 1u);
            const uint32_t below_a = a >= 32 ? 0xffffffffu : ((1u << a) - 1u);
            vis[c4] = need_mask ? (below_z & ~below_a) : 0xffffffffu;
            if (vis[c4] == 0u) hidden |= 1u << c4;
          }
#pragma unroll
          for (int c = 0; c < kBN; ++c) s[c] = (vis[c >> 5] >> (c & 31)) & 1u ? s[c] : -INFINITY;
        }
        // three-input max (FMNMX3): two new columns per instruction, four independent chains
        float mx0 = fmax3(s[0], s[1], s[2]), mx1 = fmax3(s[3], s[4], s[5]), mx2 = fmax3(s[6], s[7], s[8]), mx3 = fmax3(s[9], s[10], s[11]);
#pragma unroll
        for (int c = 12; c + 7 < kBN; c += 8) {
          mx0 = fmax3(mx0, s[c], s[c + 1]); mx1 = fmax3(mx1, s[c + 2], s[c + 3]);
          mx2 = fmax3(mx2, s[c + 4], s[c + 5]); mx3 = fmax3(mx3, s[c + 6], s[c + 7]);
        }
        mx0 = fmax3(mx0, s[kBN - 4], s[kBN - 3]); mx1 = fmax3(mx1, s[kBN - 2], s[kBN - 1]);
        const float m_new = fmax3(fmax3(mx0, mx1, mx2), mx3, m_used);
        TRACE_W(2);
        bool grow = false;
        if (m_used == -INFINITY) m_used = m_new;         // nothing accumulated yet (O row is 0 or unwritten)
        else grow = valid && (m_new - m_used) * p.scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {             // warp-uniform: tcgen05.ld/st are .sync.aligned
          // rare: O of this stream must be rescaled, so its previous P.V has to have landed.  The next
          // phase of that barrier belongs to the P.V of tile cnt + 1, which cannot be issued before this
          // thread has stored P of tile cnt, so the parity wait cannot alias.
          if (n_mine > 0) { mbar_wait(&sm.pv_done[b][(cnt - 1) & 1], ((cnt - 1) >> 1) & 1); tc_fence_after(); }
          const float alpha = grow ? ex2((m_used - m_new) * p.scale_log2) : 1.0f;
          if (grow) { l_sum *= alpha; m_used = m_new; }
          if (n_mine > 0) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              uint32_t o[32];
              tmem_ld32(t_o + lane_addr + c * 32, o);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
              tmem_st32(t_o + lane_addr + c * 32, o);
            }
          }
        }
        const float negmb = (m_used == -INFINITY) ? 0.f : -m_used * p.scale_log2;
        const uint64_t negmb2 = pack2(negmb, negmb);
        uint64_t sum_a = pack2(0.f, 0.f), sum_b = sum_a;
        // the P.V that read this P buffer two tiles ago has completed (long ago, as a rule)
        if (cnt >= 2) { mbar_wait(&sm.pv_done[b][u], ((cnt - 2) >> 1) & 1); tc_fence_after(); }
#pragma unroll
        for (int c = 0; c < kBN / 32; ++c) {
          uint32_t pk[16];
          if (hidden & (1u << c)) {                      // P = 0 without touching the MUFU
#pragma unroll
            for (int e = 0; e < 16; ++e) pk[e] = 0u;
          } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
              const uint64_t x2 = ffma2(pack2(s[c * 32 + 2 * e], s[c * 32 + 2 * e + 1]), scale2, negmb2);
              float p0, p1;
              if (((kAltOk ? kPolyMaskAlt : kPolyMaskTwoSubTiles) >> (e & 7)) & 1) {                 // three pairs of eight: FMA pipes instead of the MUFU
                exp2_poly_pair(x2, p0, p1);
              } else {
                float t0, t1;
                unpack2(x2, t0, t1);
                p0 = ex2(t0); p1 = ex2(t1);
              }
              if (e & 1) sum_b = fadd2(sum_b, pack2(p0, p1)); else sum_a = fadd2(sum_a, pack2(p0, p1));
              pk[e] = pack_bf16x2(p0, p1);
            }
          }
          tmem_st16(t_p + lane_addr + c * 16, pk);
        }
        float l0, l1;
        unpack2(fadd2(sum_a, sum_b), l0, l1);
        l_sum += l0 + l1;
        TRACE_W(3);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(&sm.p_full[b][u]);
        TRACE_W(4);
        if (tid128 == 0) TRACE_TILE(2 + 4 * b, cnt);
        ++cnt; ++n_mine;
      }
      // ---- epilogue: normalise, stage 128-byte half rows in shared memory, store coalesced ----
      if (tid128 == 0 && b == 0) TRACE(7);
      // o_full[b] completes once per piece in which the stream had key tiles (a per-P.V parity wait
      // could alias here: with Q.K^T two tiles ahead, two P.V may still be in flight)
      // what does not need the accumulator is worked out while the last P.V drains
      const float inv = l_sum > 0.f ? 1.0f / l_sum : 0.f;
      const float lse = l_sum > 0.f ? (m_used * p.scale_log2 + log2f(l_sum)) / kLog2e : -INFINITY;
      const bool whole = alt_ok || w.whole();          // an alt CTA holds ONE whole item: no partials, tickets or merges in that instance
      const int slot = 2 * (int)blockIdx.x + (w.kt_begin == 0 ? 1 : 0);
      bool do_ticket = !whole && n_rows > 0;           // a piece of a split item: publish, count, maybe merge
      if (!alt && whole && n_mine > 0) off_b[r] = (uint32_t)(out_row(p, T, w.g, b, valid ? r : 0) * (kD * 2 / 128));
      if (!alt && n_mine > 0) { mbar_wait(&sm.o_full[b], pieces_done & 1); tc_fence_after(); ++pieces_done; }
      if (tid128 == 0 && b == 0) TRACE(8);
      TRACE_E(0);
      if (alt) {
        // ---- one sub-tile, two streams (even / odd key tiles): merge them, each storing 64 columns ----
        // (the streams exchange their running maxima and row sums and work out the merge weights while their
        // last P.V drain; each waits for its own accumulator just before the second barrier)
        if (tid128 == 0) sm.alt_has[b] = n_mine > 0;
        // (an alt CTA holds ONE piece: no earlier bulk store can still be reading the staging rows)
        *reinterpret_cast<float2*>(my_stage) = make_float2(m_used, l_sum);   // exchanged through the staging rows
        bar_sync_both();
        TRACE_E(1);
        const float2 oth = *reinterpret_cast<const float2*>(sm.stage + ((b ^ 1) * kBM + r) * kStagePitch);
        const bool has0 = sm.alt_has[0] != 0, has1 = sm.alt_has[1] != 0;
        const float m0 = b ? oth.x : m_used, l0 = b ? oth.y : l_sum;
        const float m1 = b ? m_used : oth.x, l1 = b ? l_sum : oth.y;
        const float M = fmaxf(m0, m1);
        const float w0 = l0 > 0.f ? ex2((m0 - M) * p.scale_log2) : 0.f;
        const float w1 = l1 > 0.f ? ex2((m1 - M) * p.scale_log2) : 0.f;
        const float L = w0 * l0 + w1 * l1;
        const float rL = L > 0.f ? 1.0f / L : 0.f;
        const float f0 = w0 * rL, f1 = w1 * rL;
        const float lse2 = L > 0.f ? (M * p.scale_log2 + log2f(L)) / kLog2e : -INFINITY;
        if (n_mine > 0) { mbar_wait(&sm.o_full[b], pieces_done & 1); ++pieces_done; }
        bar_sync_both();                               // the exchanged values have been read (the rows may be staged over) and both accumulators are complete
        tc_fence_after();                              // the other stream's accumulator is read below, behind its thread's o_full wait
        TRACE_E(2);
        const bool full = kTmaStoreOk && T.n_tok >= p.tpt;   // the sub-tile fills its TMA box: no row beyond it may be written
        if (whole) off_b[r] = (uint32_t)(out_row(p, T, w.g, 0, valid ? r : 0) * (kD * 2 / 128));
        const uint32_t t_o0 = tmem + 256, t_o1 = tmem + 384;
#pragma unroll
        for (int c = 0; c < 2; ++c) {                  // this stream's columns [64 b + 32 c, +32)
          float o[32];
#pragma unroll
          for (int e = 0; e < 32; ++e) o[e] = 0.f;
          if (has0) {                                  // warp-uniform
            float a[32];
            tmem_ld32_f(t_o0 + lane_addr + b * 64 + c * 32, a);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] = f0 > 0.f ? a[e] * f0 : 0.f;
          }
          if (has1) {
            float a[32];
            tmem_ld32_f(t_o1 + lane_addr + b * 64 + c * 32, a);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] = f1 > 0.f ? fmaf(a[e], f1, o[e]) : o[e];
          }
          if (whole) {                                 // bf16: both chunks make one 128-byte round = half b of the tile
#pragma unroll
            for (int e = 0; e < 4; ++e)
              stage_chunk(my_stage, r, c * 4 + e,
                          make_uint4(pack_bf16x2(o[8 * e], o[8 * e + 1]), pack_bf16x2(o[8 * e + 2], o[8 * e + 3]),
                                     pack_bf16x2(o[8 * e + 4], o[8 * e + 5]), pack_bf16x2(o[8 * e + 6], o[8 * e + 7])));
            TRACE_E(3 + c);
            if (c == 1) {
              if (full) {
                AL_STAGE_ROUND_END(tma_store_3d(pmap_out, stage_b, b * 64, w.g * p.n_rep, T.q_tok0));
              } else {
                __syncwarp();
                copy_out_rows(stage_b, off_b, n_rows, tid128, reinterpret_cast<uint8_t*>(p.out) + b * 128);
                __syncwarp();
              }
              TRACE_E(5);
            }
          } else {                                     // fp32 partial (rows of sub-tile 0): one round per chunk
            if (c == 1) AL_STAGE_ROUND_BEGIN();
#pragma unroll
            for (int e = 0; e < 8; ++e)
              stage_chunk(my_stage, r, e, make_uint4(__float_as_uint(o[4 * e]), __float_as_uint(o[4 * e + 1]),
                                                     __float_as_uint(o[4 * e + 2]), __float_as_uint(o[4 * e + 3])));
            AL_STAGE_ROUND_END(bulk_store(part_round_ptr(p, slot, 0, 2 * b + c), stage_b, kBM * kStagePitch));
          }
        }
        if (whole && b == 0 && valid && p.lse) p.lse[out_row(p, T, w.g, 0, r)] = lse2;
        if (do_ticket && b == 0) p.plan.part_lse[((long long)slot * 2) * kBM + r] = valid ? lse2 : -INFINITY;
        if (do_ticket) {
          // stream 0 counts the piece for both streams: stream 1's half of the partial has to be complete
          // (performed, visible) before the barrier below lets stream 0 take the ticket
          if (tid128 == 0) { bulk_wait_all(); fence_proxy_async_all(); }
          __threadfence();
        }
        tc_fence_before();
        TRACE_E(6);
        // (no barrier, no o_empty arrival: nothing follows the CTA's one piece that could overwrite an accumulator
        // the other stream is still reading)
        TRACE_E(7);
        do_ticket = false;
      } else {
      const bool full = kTmaStoreOk && T.n_tok - b * p.tpt >= p.tpt;     // the sub-tile fills its TMA box: no row beyond it may be written
      if (n_mine == 0) {
        // nothing accumulated: no key tile of this piece concerns the sub-tile (or it is empty)
      } else if (whole) {
        // bf16 output: two rounds of 64 columns = 128 bytes per row = one 64-column half of the tile, which a full
        // sub-tile stores with ONE TMA tensor store from the staging rows (same box and swizzle as the Q loads);
        // the last, partial sub-tile of a run copies its rows out itself (off_b: set before the o_full wait)
#pragma unroll
        for (int rd = 0; rd < 2; ++rd) {
          TRACE_E(1 + 5 * rd);
          uint4 ch[8];
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            float o[32];
            tmem_ld32_f(t_o + lane_addr + rd * 64 + c * 32, o);
            tmem_wait_ld();
            if (rd == 1 && c == 1) { tc_fence_before(); mbar_arrive(&sm.o_empty[b]); }   // O_b is in registers
#pragma unroll
            for (int e = 0; e < 4; ++e)
              ch[c * 4 + e] =
                  make_uint4(pack_bf16x2(o[8 * e] * inv, o[8 * e + 1] * inv), pack_bf16x2(o[8 * e + 2] * inv, o[8 * e + 3] * inv),
                             pack_bf16x2(o[8 * e + 4] * inv, o[8 * e + 5] * inv), pack_bf16x2(o[8 * e + 6] * inv, o[8 * e + 7] * inv));
          }
          TRACE_E(2 + 5 * rd);
          if (full) {
            AL_STAGE_ROUND_BEGIN();
#pragma unroll
            for (int e = 0; e < 8; ++e) stage_chunk(my_stage, r, e, ch[e]);
            TRACE_E(3 + 5 * rd);
            AL_STAGE_ROUND_END(tma_store_3d(pmap_out, stage_b, rd * 64, w.g * p.n_rep, T.q_tok0 + b * p.tpt));
            TRACE_E(4 + 5 * rd);
          } else {
            if (rd == 0) AL_STAGE_ROUND_BEGIN();
#pragma unroll
            for (int e = 0; e < 8; ++e) stage_chunk(my_stage, r, e, ch[e]);
            __syncwarp();                              // a warp stages and copies its own 32 rows
            copy_out_rows(stage_b, off_b, n_rows, tid128, reinterpret_cast<uint8_t*>(p.out) + rd * 128);
            __syncwarp();                              // the staging rows are rewritten by the next round
          }
          TRACE_E(5 + 5 * rd);
        }
        if (valid && p.lse) p.lse[out_row(p, T, w.g, b, r)] = lse;
      } else {
        // fp32 partial: four rounds of 32 columns = 128 bytes per row, each round one 16 KB bulk store
#pragma unroll
        for (int rd = 0; rd < 4; ++rd) {
          float o[32];
          tmem_ld32_f(t_o + lane_addr + rd * 32, o);
          tmem_wait_ld();
          if (rd == 3) { tc_fence_before(); mbar_arrive(&sm.o_empty[b]); }
          AL_STAGE_ROUND_BEGIN();
#pragma unroll
          for (int e = 0; e < 8; ++e)
            stage_chunk(my_stage, r, e, make_uint4(__float_as_uint(o[4 * e] * inv), __float_as_uint(o[4 * e + 1] * inv),
                                                   __float_as_uint(o[4 * e + 2] * inv), __float_as_uint(o[4 * e + 3] * inv)));
          AL_STAGE_ROUND_END(bulk_store(part_round_ptr(p, slot, b, rd), stage_b, kBM * kStagePitch));
        }
      }
      if (do_ticket) {
        p.plan.part_lse[((long long)slot * 2 + b) * kBM + r] = (valid && n_mine > 0) ? lse : -INFINITY;
        __threadfence();
      }
      }
      if (tid128 == 0 && b == 0) TRACE(9);
      if (do_ticket) {
        bar_sync_stream(b);
        if (tid128 == 0 && b == 0) TRACE(10);
        if (tid128 == 0) {
          // the bulk stores of this stream's partial have completed (in alt mode stream 1's too: see below)
          bulk_wait_all();
          fence_proxy_async_all();
          __threadfence();
          // pieces of this item live on consecutive CTAs c0..c1 (from the plan): a piece that does not
          // start its item is this CTA's first piece, one that does not finish it is its last
          const int c0 = w.kt_begin > 0 ? w.first_c0 : w.last_c0;
          const int c1 = w.kt_begin > 0 ? w.first_c1 : w.last_c1;
          int* counter = p.plan.counters + 2 * w.item() + b;
          const int old = atomicAdd(counter, 1);
          const bool last = old == c1 - c0;
          if (last) *counter = 0;                      // every piece has arrived: leave the counter clean
          sm.ticket[b][0] = last ? 1 : 0; sm.ticket[b][1] = c0; sm.ticket[b][2] = c1;
        }
        bar_sync_stream(b);
        if (sm.ticket[b][0]) {
          __threadfence();
          if (tid128 == 0 && b == 0) TRACE(11);
          merge_item(p, T, w.g, b, sm.ticket[b][1], sm.ticket[b][2], tid128);
          if (tid128 == 0 && b == 0) TRACE(12);
        }
        bar_sync_stream(b);                            // ticket is reused by the next piece
      }
    }
    if (tid128 == 0) bulk_wait_read_all();             // the staging rows must outlive the bulk stores that read them (their writes complete with the grid)
  }
}

// ---------------------------------------------------------------------------------------------
// self-planned launches: no plan kernel in front of the attention
// ---------------------------------------------------------------------------------------------
// Small calls (at most 32 lanes; by the host's bounds every item has a CTA of its own and no item is long
// enough for the plan kernel to cut it -- self_plan_ok below) take the whole-item plan whatever the descriptors hold,
// and CTA c = item (tile c / n_kv, kv-head c % n_kv) needs nothing but its own tile.  One warp derives it
// from the lane descriptors in the prologue, one lane per thread: the arithmetic of lane_plan_kernel's
// whole-item branch (runs -> tiles per run -> the tile's lanes) with ballots and warp reductions in place
// of the block scans.  It costs the one global read the record load would cost, and the 5-6 us plan launch
// that such a call cannot hide behind anything goes away.
__device__ __noinline__ void self_plan_record(const al_lane_desc* __restrict__ lanes, int n_lanes, int n_kv, int tpt,
                                              int grid, int cta, CtaRec* out) {
  const unsigned full = 0xffffffffu;
  const int i = threadIdx.x & 31;
  const bool has = i < n_lanes;
  int grp = 0, kb = 0, pl = 0, qs = 0, ql = 0;
  if (has) {
    const int2* d = reinterpret_cast<const int2*>(lanes + i);
    const int2 a = __ldcg(d), b = __ldcg(d + 1), c = __ldcg(d + 2);
    grp = a.x; kb = a.y; pl = b.x; qs = b.y; ql = c.x;
  }
  const int qe = qs + ql;
  const int p_grp = __shfl_up_sync(full, grp, 1), p_kb = __shfl_up_sync(full, kb, 1), p_qe = __shfl_up_sync(full, qe, 1);
  const bool start = has && (i == 0 || !(p_grp == grp && p_kb == kb && p_qe == qs));
  const unsigned starts = __ballot_sync(full, start);
  // the run of lane i: [l0, l1) = [last start at or below i, next start above i)
  const unsigned upto = (2u << i) - 1u;
  const int l0 = has ? 31 - __clz(starts & upto) : 0;
  const unsigned above = starts & ~upto;
  const int l1 = has ? (above ? __ffs(above) - 1 : n_lanes) : 1;
  const int run_q1 = __shfl_sync(full, qe, l1 - 1);
  const int span = start ? max(0, run_q1 - qs) : 0;
  (void)l0;
  const int tiles2 = __reduce_add_sync(full, start ? ceil_div(span, 2 * tpt) : 0);
  const int tile_tok = (tiles2 > 0 && 4 * tiles2 * n_kv <= grid) ? tpt : 2 * tpt;   // as lane_plan_kernel
  const int my_tiles = start ? ceil_div(span, tile_tok) : 0;
  int incl = my_tiles;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int y = __shfl_up_sync(full, incl, off);
    if (i >= off) incl += y;
  }
  const int base = incl - my_tiles, n_tiles = __shfl_sync(full, incl, 31);
  const int t = cta / n_kv, g = cta - t * n_kv;
  CtaRec C{};
  C.first_c0 = C.first_c1 = C.last_c0 = C.last_c1 = cta;
  C.pad = cta;
  C.flags = kCtaAlt;                                         // idle unless the CTA has a tile
  if (t < n_tiles) {                                         // warp-uniform
    const unsigned owner = __ballot_sync(full, start && base <= t && t < base + my_tiles);
    const int o = __ffs(owner) - 1;                          // first lane of the run that holds tile t
    const int r_l1 = __shfl_sync(full, l1, o), r_base = __shfl_sync(full, base, o);
    const int r_q0 = __shfl_sync(full, qs, o), r_q1 = __shfl_sync(full, run_q1, o), r_kb = __shfl_sync(full, kb, o);
    TileRec T;
    T.q_tok0 = r_q0 + (t - r_base) * tile_tok;
    T.n_tok = min(tile_tok, r_q1 - T.q_tok0);
    T.kv_base_row = r_kb;
    const int end = T.q_tok0 + T.n_tok;
    const bool in_run = has && i >= o && i < r_l1;
    const int lf = 31 - __clz(__ballot_sync(full, in_run && qs <= T.q_tok0));   // lane that holds the tile's first token
    const bool member = in_run && i >= lf && qs < end;
    T.lane_first = lf; T.lane_count = __popc(__ballot_sync(full, member));
    T.kv_len_max = __reduce_max_sync(full, member ? pl : 0);
    T.kv_len_min = __reduce_min_sync(full, member ? pl : 0x7fffffff);
    T.lk0 = __reduce_min_sync(full, member ? qs : 0x7fffffff);
    T.lk1 = __reduce_max_sync(full, member ? qe : 0);
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const int t0 = T.q_tok0 + b * tpt, t1 = min(t0 + tpt, end);
      const bool hit = member && qs < t1 && qe > t0;
      T.sub_lk0[b] = __reduce_min_sync(full, hit ? qs : 0x7fffffff);
      T.sub_lk1[b] = __reduce_max_sync(full, hit ? qe : 0);
    }
    T.n_pref_tiles = ceil_div(T.kv_len_max, kBN);
    T.n_key_tiles = T.n_pref_tiles + ceil_div(T.lk1 - T.lk0, kBN);
    T.kt_off = 0;                                            // the CTA's steps are counted from its own tile
    C.f_begin = g * T.n_key_tiles; C.f_end = C.f_begin + T.n_key_tiles;
    C.tile0 = t;
    C.flags = kCtaActive | (T.n_tok <= tpt ? kCtaAlt : 0);     // one sub-tile: both streams work on it (alt instance)
    C.first = T;
  }
  if (i == 0) *out = C;
}

// kSelfPlan: the launch has no plan (self_plan_record).  Two kernels rather than a switch in one: the
// plan-reading kernel keeps the prologue it had (its schedule is sensitive to anything added around it), and
// each kernel lays out first the instance of the roles its launches use most.
template <bool kSelfPlan>
__global__ void __launch_bounds__(kThreads, 1)
lane_attention_umma_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_knew,
                           const __grid_constant__ CUtensorMap map_vnew, const __grid_constant__ CUtensorMap map_kc,
                           const __grid_constant__ CUtensorMap map_vc, const __grid_constant__ CUtensorMap map_out,
                           const AttnParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  AttnSmem& sm = *reinterpret_cast<AttnSmem*>(smem_raw);
  // the shuffle tells the compiler that `warp` is warp-uniform: the role branches and everything derived
  // from it (stream index, TMEM and shared-memory descriptors) then live in uniform registers
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  TRACE_RESET();
  if (threadIdx.x == 0) {
    if (smem_u32(smem_raw) & 1023u) __trap();          // the 128-byte swizzle atoms need 1024-byte alignment
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 2);       // the *_empty barriers expect two arrivals (one per issuing warp, or two from the one that issues for both streams)
    for (int s = 0; s < kStagesK; ++s) { mbar_init(&sm.k_full[s], 1); mbar_init(&sm.k_empty[s], 2); }
    for (int s = 0; s < kStagesV; ++s) { mbar_init(&sm.v_full[s], 1); mbar_init(&sm.v_empty[s], 2); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(&sm.s_full[b], 1); mbar_init(&sm.s_free[b], 128);
      for (int u = 0; u < 2; ++u) { mbar_init(&sm.p_full[b][u], 128); mbar_init(&sm.pv_done[b][u], 1); }
      mbar_init(&sm.o_full[b], 1); mbar_init(&sm.o_empty[b], 128);
    }
    fence_barrier_init();
    prefetch_tensormap(&map_q); prefetch_tensormap(&map_knew); prefetch_tensormap(&map_vnew);
    prefetch_tensormap(&map_kc); prefetch_tensormap(&map_vc); prefetch_tensormap(&map_out);
  }
  if (warp == 1) tmem_alloc<512>(&sm.tmem_base);
  // programmatic dependent launch: everything above overlapped the previous kernel in the stream (the
  // plan, or the previous layer); its memory is visible after the wait.  The next launch in the stream
  // that opts in (the next layer) may then begin its own prologue as SMs free up.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // the CTA's plan record: the one global read on the way to the first TMA load, in flight under the TMEM
  // allocation and the barrier initialisation of the other warps
  if constexpr (kSelfPlan) {
    if (warp == 2) self_plan_record(p.lanes, p.n_lanes, p.n_kv_heads, p.tpt, (int)gridDim.x, (int)blockIdx.x, &sm.cta);
  } else {
    if (warp == 2 && lane < (int)(sizeof(CtaRec) / 16))
      reinterpret_cast<uint4*>(&sm.cta)[lane] = __ldcg(reinterpret_cast<const uint4*>(p.plan.ctas + blockIdx.x) + lane);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  // TMEM columns: S of stream b at 64 b; P of stream b, buffer u at 128 + 64 b + 32 u; O of stream b at 256 + 128 b
  // Two instances of the roles: one for CTAs whose (single, whole) item has ONE sub-tile, which both streams
  // work on (kCtaAlt in the CTA's record; `alt` is a compile-time constant there), one for everything else.  The
  // instance laid out FIRST runs measurably faster inside a step (cfg5 plan + attention 67.5 us with the
  // general instance first, 71.5 us with it second; cfg4 620 us against 634 us per 32 layers the other way
  // round): the plan-reading kernel gives the throughput configuration the first place, the self-planned one
  // (small calls: one sub-tile as a rule) the alt instance.
  if constexpr (kSelfPlan) {
    if (sm.cta.flags & kCtaAlt) attn_roles<true>(sm, p, &map_q, &map_knew, &map_vnew, &map_kc, &map_vc, &map_out, tmem, warp, lane);
    else attn_roles<false>(sm, p, &map_q, &map_knew, &map_vnew, &map_kc, &map_vc, &map_out, tmem, warp, lane);
  } else {
    if (!(sm.cta.flags & kCtaAlt)) attn_roles<false>(sm, p, &map_q, &map_knew, &map_vnew, &map_kc, &map_vc, &map_out, tmem, warp, lane);
    else attn_roles<true>(sm, p, &map_q, &map_knew, &map_vnew, &map_kc, &map_vc, &map_out, tmem, warp, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) TRACE(13);
  if (warp == 1) { __syncwarp(); tmem_dealloc<512>(tmem); }
  if (threadIdx.x == 32) TRACE(14);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
Bounds bounds_for(const al_attn_shape* s, int n_lanes, int total_q_rows, int n_sms) {
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  const int tpt = kBM / n_rep;
  Bounds b;
  b.max_tiles = ceil_div(total_q_rows, 2 * tpt) + n_lanes;   // (one-sub-tile plans have at most grid / (2 n_kv) tiles)
  if (b.max_tiles < kMaxCtas) b.max_tiles = kMaxCtas;
  b.grid = n_sms < kMaxCtas ? n_sms : kMaxCtas;
  return b;
}

// Calls whose plan every CTA can derive for itself (self_plan_record): one lane per thread of a warp; every
// item a CTA of its own even if every lane were a run of its own and every tile took one sub-tile; and no
// item longer than kSelfPlanMaxSteps key tiles, for which lane_plan_kernel takes the whole-item plan whatever
// the descriptors hold (s_max_nk <= kMinPiece + kSplitCost) -- so the self-planned record IS the plan kernel's.
// Decided from the host's bounds alone: al_lane_plan and al_lane_attention_planned, given the same bounds,
// agree without talking to each other.
constexpr int kSelfPlanMaxSteps = kMinPiece + kSplitCost;
bool self_plan_ok(const al_handle* h, const al_attn_shape* s, int n_lanes, int total_q_rows, int max_prefix_len,
                  const Bounds& b) {
  if (!h->self_plan || n_lanes > 32) return false;
  const int tpt = kBM / (s->n_q_heads / s->n_kv_heads);
  const long long tiles = (long long)ceil_div(total_q_rows, tpt) + n_lanes - 1;
  if (tiles * s->n_kv_heads > b.grid) return false;
  return ceil_div(max_prefix_len, kBN) + ceil_div(total_q_rows, kBN) <= kSelfPlanMaxSteps;
}

struct WsLayout {
  size_t hdr, tiles, ctas, bounds, counters, order, part_lse, part_o, total;
};
WsLayout ws_layout(const al_attn_shape* s, const Bounds& b) {
  WsLayout L;
  size_t off = 0;
  auto take = [&](size_t n) { size_t o = off; off = al_round_up(off + n, 256); return o; };
  L.hdr = take(sizeof(PlanHeader));
  L.tiles = take(sizeof(TileRec) * (size_t)b.max_tiles);
  L.ctas = take(sizeof(CtaRec) * (size_t)b.grid);
  L.bounds = take(sizeof(int) * (size_t)(b.grid + 1));
  L.counters = take(sizeof(int) * (size_t)b.max_tiles * s->n_kv_heads * 2);
  L.order = take(sizeof(int) * (size_t)b.max_tiles * s->n_kv_heads);
  L.part_lse = take(sizeof(float) * (size_t)2 * b.grid * 2 * kBM);
  L.part_o = take(sizeof(float) * (size_t)2 * b.grid * 2 * kBM * kD);
  L.total = off;
  return L;
}

constexpr int kSmsForBounds = kMaxCtas;   // workspace sizing when no handle is at hand (>= SMs of any B200)

Plan plan_in(void* workspace, const WsLayout& L) {
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  Plan plan;
  plan.hdr = reinterpret_cast<PlanHeader*>(ws + L.hdr);
  plan.tiles = reinterpret_cast<TileRec*>(ws + L.tiles);
  plan.ctas = reinterpret_cast<CtaRec*>(ws + L.ctas);
  plan.bounds = reinterpret_cast<int*>(ws + L.bounds);
  plan.counters = reinterpret_cast<int*>(ws + L.counters);
  plan.order = reinterpret_cast<int*>(ws + L.order);
  plan.part_lse = reinterpret_cast<float*>(ws + L.part_lse);
  plan.part_o = reinterpret_cast<float*>(ws + L.part_o);
  return plan;
}

al_status make_map_3d(const al_handle* h, CUtensorMap* map, const void* base, uint64_t d0, uint64_t d1, uint64_t d2,
                      uint64_t stride1_bytes, uint64_t stride2_bytes, uint32_t b0, uint32_t b1, uint32_t b2) {
  const cuuint64_t dims[3] = {d0, d1, d2};
  const cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
  const cuuint32_t box[3] = {b0, b1, b2};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = h->encode_tiled(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box,
                               estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) AL_FAIL(AL_ERR_CUDA, "cuTensorMapEncodeTiled(3d) failed: %d", (int)r);
  return AL_OK;
}

al_status check_plan_bounds(const al_attn_shape* s, int n_lanes, const Bounds& b) {
  (void)s;
  if (n_lanes > kMaxPlanLanes) AL_FAIL(AL_ERR_UNSUPPORTED, "al_lane_attention: more than %d lanes", kMaxPlanLanes);
  if (b.max_tiles > kMaxPlanTiles)
    AL_FAIL(AL_ERR_UNSUPPORTED, "al_lane_attention: more than %d query tiles (total_q_rows too large)", kMaxPlanTiles);
  return AL_OK;
}

}  // namespace

bool al_attention_umma_supported(const al_attn_shape* s) {
  if (s->dtype != AL_BF16 || s->head_dim != kD) return false;
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  return n_rep >= 1 && n_rep <= kBM;
}

al_status al_attention_umma_check(const al_handle* h, const al_attn_shape* s, int n_lanes, int total_q_rows) {
  return check_plan_bounds(s, n_lanes, bounds_for(s, n_lanes, total_q_rows, h->sm_count));
}

size_t al_attention_umma_workspace_bytes(const al_handle* h, const al_attn_shape* s, int n_lanes, int total_q_rows,
                                         int max_prefix_len) {
  (void)max_prefix_len;
  const Bounds b = bounds_for(s, n_lanes, total_q_rows, h ? h->sm_count : kSmsForBounds);
  return ws_layout(s, b).total;
}

al_status al_launch_plan_umma(const al_handle* h, const al_attn_shape* s, const al_lane_desc* lanes, int n_lanes,
                              int total_q_rows, int max_prefix_len, void* workspace, size_t workspace_bytes,
                              cudaStream_t st) {
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  const int tpt = kBM / n_rep;
  const Bounds b = bounds_for(s, n_lanes, total_q_rows, h->sm_count);
  al_status rc = check_plan_bounds(s, n_lanes, b);
  if (rc != AL_OK) return rc;
  const WsLayout L = ws_layout(s, b);
  if (workspace_bytes < L.total) AL_FAIL(AL_ERR_WORKSPACE, "al_lane_plan: workspace %zu < %zu", workspace_bytes, L.total);
  if (self_plan_ok(h, s, n_lanes, total_q_rows, max_prefix_len, b)) return AL_OK;   // the attention CTAs plan for themselves
  lane_plan_kernel<<<1, kPlanThreads, 0, st>>>(lanes, n_lanes, s->n_kv_heads, tpt, b, plan_in(workspace, L));
  AL_CUDA_OK(cudaGetLastError());
  h->launches += 1;
  return AL_OK;
}

al_status al_launch_attention_umma(const al_handle* h, const al_attn_shape* s, float scale, const void* q,
                                   const void* k_new, const void* v_new, const void* k_cache, const void* v_cache,
                                   const al_lane_desc* lanes, int n_lanes, int total_q_rows, int max_prefix_len,
                                   void* out, float* lse, void* workspace, size_t workspace_bytes, cudaStream_t st) {
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  const int tpt = kBM / n_rep;
  const Bounds b = bounds_for(s, n_lanes, total_q_rows, h->sm_count);
  al_status rc = check_plan_bounds(s, n_lanes, b);
  if (rc != AL_OK) return rc;
  const WsLayout L = ws_layout(s, b);
  if (workspace_bytes < L.total) AL_FAIL(AL_ERR_WORKSPACE, "al_lane_attention: workspace %zu < %zu", workspace_bytes, L.total);

  CUtensorMap mq, mkn, mvn, mkc, mvc, mo;
  const uint64_t T = (uint64_t)total_q_rows, Hq = (uint64_t)s->n_q_heads, Hkv = (uint64_t)s->n_kv_heads;
  const uint64_t rowb = kD * 2;
  if ((rc = make_map_3d(h, &mq, q, kD, Hq, T, rowb, Hq * rowb, 64, (uint32_t)n_rep, (uint32_t)tpt)) != AL_OK) return rc;
  // the output has the layout of Q: a full sub-tile's 64-column half is stored with the box it was loaded with
  if ((rc = make_map_3d(h, &mo, out, kD, Hq, T, rowb, Hq * rowb, 64, (uint32_t)n_rep, (uint32_t)tpt)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mkn, k_new, kD, Hkv, T, rowb, Hkv * rowb, 64, 1, kBN)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mvn, v_new, kD, Hkv, T, rowb, Hkv * rowb, 64, 1, kBN)) != AL_OK) return rc;
  // a group with no prefix never touches the cache maps; encode them over k_new when there is no cache
  const uint64_t crows = s->cache_rows > 0 && k_cache ? (uint64_t)s->cache_rows : 1;
  const void* kc = (s->cache_rows > 0 && k_cache) ? k_cache : k_new;
  const void* vc = (s->cache_rows > 0 && v_cache) ? v_cache : v_new;
  if ((rc = make_map_3d(h, &mkc, kc, kD, crows, Hkv, rowb, crows * rowb, 64, kBN, 1)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mvc, vc, kD, crows, Hkv, rowb, crows * rowb, 64, kBN, 1)) != AL_OK) return rc;

  AttnParams p;
  p.lanes = lanes; p.plan = plan_in(workspace, L); p.out = static_cast<__nv_bfloat16*>(out); p.lse = lse;
  p.n_q_heads = s->n_q_heads; p.n_kv_heads = s->n_kv_heads; p.n_rep = n_rep; p.tpt = tpt;
  p.scale_log2 = scale * kLog2e;
  p.n_lanes = n_lanes;
  const bool self_plan = self_plan_ok(h, s, n_lanes, total_q_rows, max_prefix_len, b);
  p.q_box_bytes = (uint32_t)(2 * tpt * n_rep * 64 * 2);
  const size_t smem = sizeof(AttnSmem);
  AL_CUDA_OK(cudaFuncSetAttribute(lane_attention_umma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  AL_CUDA_OK(cudaFuncSetAttribute(lane_attention_umma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)b.grid);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.wait in the kernel
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (self_plan) AL_CUDA_OK(cudaLaunchKernelEx(&cfg, lane_attention_umma_kernel<true>, mq, mkn, mvn, mkc, mvc, mo, p));
  else AL_CUDA_OK(cudaLaunchKernelEx(&cfg, lane_attention_umma_kernel<false>, mq, mkn, mvn, mkc, mvc, mo, p));
  h->launches += 1;
  return AL_OK;
}
