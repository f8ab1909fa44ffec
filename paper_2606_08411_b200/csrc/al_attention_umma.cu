// K1 lane_attention (bf16, head_dim 128) on the 5th-generation tensor cores -- al_lane_attention's
// main path (Eq.2-3: each lane attends to its prefix state kappa_l and to its
// own rows; L168-172 Eq.11: lanes of one shared-prefix group are evaluated in one batched call).
//
// Work decomposition (built ON DEVICE from the lane descriptors by lane_plan_kernel, so the call is
// graph-replayable with new lanes):
//   run    = maximal sequence of lanes adjacent in the array, of one group, contiguous in q_start
//   tile   = up to tpt = floor(128 / n_rep) consecutive tokens of a run; with the n_rep q-heads of a
//            kv-head stacked under every token it is a 128-row M tile of the tensor core
//   keys   = [prefix key tiles of 128 cache rows] ++ [local key tiles of 128 K_new rows covering the
//            lanes that intersect the tile]; every row masks what its own lane may not see
//   work   = (tile, kv-head, contiguous range of key tiles); a tile whose key range is split over
//            several CTAs (to fill the SMs when heads x tiles are few) leaves fp32 partials + LSE in
//            the workspace and lane_combine_kernel merges them.
// All CTAs that share (group, kv-head) read the same K/V tiles: HBM sees them once, L2 serves the
// rest -- "the prefix is read once per lane group" (BASELINE north_star).
//
// Main kernel, persistent, 192 threads, warp-specialised:
//   warp 0     TMA producer: Q tile once per work item, K and V tiles through a 3-stage ring
//   warp 1     MMA issuer (one elected lane): S = Q.K^T (SS form) into a double-buffered TMEM tile,
//              O += P.V with P read from TMEM (TS form) and V MN-major in shared memory
//   warps 2-5  online softmax, one thread per row: tcgen05.ld S, mask, running max with lazy
//              rescaling of O (only when the max grows by more than 2^8), exp2, bf16 P back into
//              the TMEM columns of S, row sums in fp32; then the epilogue (normalise, store)
#include <cuda_bf16.h>

#include "al_internal.h"
#include "al_ptx.cuh"

using namespace alptx;

namespace {

constexpr int kBM = 128;                   // stacked query rows per tile
constexpr int kBN = 128;                   // keys per key tile
constexpr int kD = 128;                    // head_dim
constexpr int kStages = 3;                 // K/V ring depth
constexpr int kHalfBytes = 128 * 64 * 2;   // [128 rows][64 bf16] = one 128-byte-swizzled half tile
constexpr int kTileBytes = 2 * kHalfBytes;
constexpr int kThreads = 192;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: P <= 2^8 between rescales
constexpr int kMaxPlanLanes = 2048;

struct __align__(16) TileRec {
  int q_tok0, n_tok;         // first packed token row, tokens in the tile
  int kv_base_row;           // cache row of prefix key 0
  int kv_len_max, kv_len_min;// largest / smallest prefix_len among the lanes of the tile
  int lk0, lk1;              // local keys: packed rows [lk0, lk1) of K_new / V_new
  int lane_first, lane_count;
  int n_pref_tiles, n_key_tiles;
  int n_splits, work_base, part_base;   // part_base: first partial slot (-1 when not split)
  int pad0, pad1;
};
struct __align__(16) WorkRec {
  int tile, g, kt_begin, kt_end;
  int part_slot, split, pad0, pad1;
};
struct PlanHeader {
  int n_tiles, n_work, n_part, chunk;
};

struct Plan {
  PlanHeader* hdr;
  TileRec* tiles;
  WorkRec* work;
  float* part_o;     // [n_part][128][128]
  float* part_lse;   // [n_part][128]
};

struct Bounds {
  int max_tiles, max_work, max_part;
};

__host__ __device__ inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// ---------------------------------------------------------------------------------------------
// plan: lanes -> tiles -> work items.  One CTA; sizes are tiny (lanes <= 2048, tiles <= a few 100).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
lane_plan_kernel(const al_lane_desc* __restrict__ lanes, int n_lanes, int n_kv_heads, int tpt, int n_sms,
                 Bounds bounds, Plan plan) {
  __shared__ int s_run_of_lane_start[kMaxPlanLanes];   // 1 if lane i starts a run
  __shared__ int s_run_tile_base[kMaxPlanLanes + 1];   // per run: first tile
  __shared__ int s_run_lane0[kMaxPlanLanes + 1];       // per run: first lane (sentinel n_lanes at the end)
  __shared__ int s_n_runs, s_n_tiles, s_total_kt, s_chunk, s_n_work, s_n_part;
  const int tid = threadIdx.x;

  for (int i = tid; i < n_lanes; i += blockDim.x) {
    int start = 1;
    if (i > 0) {
      const al_lane_desc a = lanes[i - 1], b = lanes[i];
      start = !(a.group_id == b.group_id && a.kv_base_row == b.kv_base_row && a.q_start + a.q_len == b.q_start);
    }
    s_run_of_lane_start[i] = start;
  }
  __syncthreads();
  if (tid == 0) {
    int n_runs = 0, n_tiles = 0;
    for (int i = 0; i < n_lanes; ++i)
      if (s_run_of_lane_start[i]) s_run_lane0[n_runs++] = i;
    s_run_lane0[n_runs] = n_lanes;
    for (int r = 0; r < n_runs; ++r) {
      const int l0 = s_run_lane0[r], l1 = s_run_lane0[r + 1];
      const int tok0 = lanes[l0].q_start, tok1 = lanes[l1 - 1].q_start + lanes[l1 - 1].q_len;
      s_run_tile_base[r] = n_tiles;
      n_tiles += ceil_div(tok1 - tok0, tpt);
    }
    s_run_tile_base[n_runs] = n_tiles;
    s_n_runs = n_runs;
    s_n_tiles = min(n_tiles, bounds.max_tiles);
    s_total_kt = 0;
  }
  __syncthreads();
  const int n_runs = s_n_runs, n_tiles = s_n_tiles;

  // tiles (one thread each)
  for (int t = tid; t < n_tiles; t += blockDim.x) {
    int r = 0;
    while (s_run_tile_base[r + 1] <= t) ++r;
    const int l0 = s_run_lane0[r], l1 = s_run_lane0[r + 1];
    const int run_tok0 = lanes[l0].q_start, run_tok1 = lanes[l1 - 1].q_start + lanes[l1 - 1].q_len;
    TileRec T;
    T.q_tok0 = run_tok0 + (t - s_run_tile_base[r]) * tpt;
    T.n_tok = min(tpt, run_tok1 - T.q_tok0);
    T.kv_base_row = lanes[l0].kv_base_row;
    T.kv_len_max = 0; T.kv_len_min = 0x7fffffff; T.lk0 = 0x7fffffff; T.lk1 = 0; T.lane_first = -1; T.lane_count = 0;
    for (int l = l0; l < l1; ++l) {
      const al_lane_desc L = lanes[l];
      if (L.q_start < T.q_tok0 + T.n_tok && L.q_start + L.q_len > T.q_tok0) {
        if (T.lane_first < 0) T.lane_first = l;
        T.lane_count = l - T.lane_first + 1;
        T.kv_len_max = max(T.kv_len_max, L.prefix_len);
        T.kv_len_min = min(T.kv_len_min, L.prefix_len);
        T.lk0 = min(T.lk0, L.q_start);
        T.lk1 = max(T.lk1, L.q_start + L.q_len);
      }
    }
    T.n_pref_tiles = ceil_div(T.kv_len_max, kBN);
    T.n_key_tiles = T.n_pref_tiles + ceil_div(T.lk1 - T.lk0, kBN);
    T.n_splits = 1; T.work_base = 0; T.part_base = -1; T.pad0 = T.pad1 = 0;
    plan.tiles[t] = T;
    atomicAdd(&s_total_kt, T.n_key_tiles);
  }
  __syncthreads();
  // split policy: chunk = key tiles per work item so that the busiest SM gets ceil(total / SMs)
  if (tid == 0) {
    const long long total = (long long)s_total_kt * n_kv_heads;
    int chunk = (int)((total + n_sms - 1) / n_sms);
    if (chunk < 1) chunk = 1;
    int n_work = 0, n_part = 0;
    for (int t = 0; t < n_tiles; ++t) {
      TileRec& T = plan.tiles[t];
      int ns = ceil_div(T.n_key_tiles, chunk);
      if (ns > 1 && n_part + ns * n_kv_heads > bounds.max_part) ns = 1;       // never outgrow the workspace
      T.n_splits = ns;
      T.work_base = n_work;
      T.part_base = ns > 1 ? n_part : -1;
      n_work += ns * n_kv_heads;
      if (ns > 1) n_part += ns * n_kv_heads;
    }
    s_chunk = chunk; s_n_work = n_work; s_n_part = n_part;
    plan.hdr->n_tiles = n_tiles; plan.hdr->n_work = n_work; plan.hdr->n_part = n_part; plan.hdr->chunk = chunk;
  }
  __syncthreads();
  __threadfence_block();
  // work items (one thread each): index = work_base + g * n_splits + split
  for (int t = 0; t < n_tiles; ++t) {
    const TileRec T = plan.tiles[t];
    const int n = T.n_splits * n_kv_heads;
    for (int j = tid; j < n; j += blockDim.x) {
      const int g = j / T.n_splits, sp = j - g * T.n_splits;
      WorkRec W;
      W.tile = t; W.g = g;
      // even partition of the key tiles over the splits
      W.kt_begin = (int)((long long)T.n_key_tiles * sp / T.n_splits);
      W.kt_end = (int)((long long)T.n_key_tiles * (sp + 1) / T.n_splits);
      W.part_slot = T.part_base < 0 ? -1 : T.part_base + j;
      W.split = sp; W.pad0 = W.pad1 = 0;
      plan.work[T.work_base + j] = W;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// main kernel
// ---------------------------------------------------------------------------------------------
struct AttnSmem {
  alignas(1024) uint8_t q[2][kHalfBytes];
  alignas(1024) uint8_t k[kStages][2][kHalfBytes];
  alignas(1024) uint8_t v[kStages][2][kHalfBytes];
  uint64_t q_full, q_empty;
  uint64_t k_full[kStages], v_full[kStages], kv_empty[kStages];
  uint64_t s_full[2], p_full[2];
  uint64_t pv_done, o_empty;
  uint32_t tmem_base;
};

struct AttnParams {
  const al_lane_desc* lanes;
  Plan plan;
  __nv_bfloat16* out;
  float* lse;
  int n_q_heads, n_kv_heads, n_rep;
  uint32_t q_box_bytes;
  float scale_log2;
};

__device__ __forceinline__ void tmem_ld32_f(uint32_t taddr, float* dst) {
  uint32_t r[32];
  tmem_ld32(taddr, r);
#pragma unroll
  for (int i = 0; i < 32; ++i) dst[i] = __uint_as_float(r[i]);
}

__global__ void __launch_bounds__(kThreads, 1)
lane_attention_umma_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_knew,
                           const __grid_constant__ CUtensorMap map_vnew, const __grid_constant__ CUtensorMap map_kc,
                           const __grid_constant__ CUtensorMap map_vc, const AttnParams p) {
  extern __shared__ uint8_t smem_raw[];
  AttnSmem& sm = *reinterpret_cast<AttnSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 1);
    for (int s = 0; s < kStages; ++s) { mbar_init(&sm.k_full[s], 1); mbar_init(&sm.v_full[s], 1); mbar_init(&sm.kv_empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&sm.s_full[b], 1); mbar_init(&sm.p_full[b], 128); }
    mbar_init(&sm.pv_done, 1); mbar_init(&sm.o_empty, 128);
    fence_barrier_init();
    prefetch_tensormap(&map_q); prefetch_tensormap(&map_knew); prefetch_tensormap(&map_vnew);
    prefetch_tensormap(&map_kc); prefetch_tensormap(&map_vc);
  }
  if (warp == 1) tmem_alloc<512>(&sm.tmem_base);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  const uint32_t t_s[2] = {tmem, tmem + 128};
  const uint32_t t_o = tmem + 256;
  const int n_work = p.plan.hdr->n_work;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      uint32_t kv_it = 0, item_it = 0;
      for (int w = blockIdx.x; w < n_work; w += gridDim.x, ++item_it) {
        const WorkRec W = p.plan.work[w];
        const TileRec T = p.plan.tiles[W.tile];
        mbar_wait(&sm.q_empty, (item_it & 1) ^ 1);
        mbar_arrive_expect_tx(&sm.q_full, p.q_box_bytes);   // the box is tpt*n_rep (<= 128) rows per half
        tma_load_3d(sm.q[0], &map_q, &sm.q_full, 0, W.g * p.n_rep, T.q_tok0);
        tma_load_3d(sm.q[1], &map_q, &sm.q_full, 64, W.g * p.n_rep, T.q_tok0);
        for (int kt = W.kt_begin; kt < W.kt_end; ++kt, ++kv_it) {
          const int s = kv_it % kStages;
          const uint32_t ph = (kv_it / kStages) & 1;
          mbar_wait(&sm.kv_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&sm.k_full[s], kTileBytes);
          if (kt < T.n_pref_tiles) {
            const int row = T.kv_base_row + kt * kBN;
            tma_load_3d(sm.k[s][0], &map_kc, &sm.k_full[s], 0, row, W.g);
            tma_load_3d(sm.k[s][1], &map_kc, &sm.k_full[s], 64, row, W.g);
            mbar_arrive_expect_tx(&sm.v_full[s], kTileBytes);
            tma_load_3d(sm.v[s][0], &map_vc, &sm.v_full[s], 0, row, W.g);
            tma_load_3d(sm.v[s][1], &map_vc, &sm.v_full[s], 64, row, W.g);
          } else {
            const int row = T.lk0 + (kt - T.n_pref_tiles) * kBN;
            tma_load_3d(sm.k[s][0], &map_knew, &sm.k_full[s], 0, W.g, row);
            tma_load_3d(sm.k[s][1], &map_knew, &sm.k_full[s], 64, W.g, row);
            mbar_arrive_expect_tx(&sm.v_full[s], kTileBytes);
            tma_load_3d(sm.v[s][0], &map_vnew, &sm.v_full[s], 0, W.g, row);
            tma_load_3d(sm.v[s][1], &map_vnew, &sm.v_full[s], 64, W.g, row);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      const uint32_t idesc_qk = make_idesc_bf16(kBM, kBN, 0, 0);
      const uint32_t idesc_pv = make_idesc_bf16(kBM, kD, 0, 1);
      uint32_t kv_it = 0, sp_it = 0, item_it = 0;
      for (int w = blockIdx.x; w < n_work; w += gridDim.x, ++item_it) {
        const WorkRec W = p.plan.work[w];
        const TileRec T = p.plan.tiles[W.tile];
        const int n = W.kt_end - W.kt_begin;
        mbar_wait(&sm.q_full, item_it & 1);
        tc_fence_after();
        const uint32_t kv_base_it = kv_it, sp_base_it = sp_it;
        for (int i = 0; i <= n; ++i) {
          if (i < n) {
            const uint32_t it = kv_base_it + i;
            const int s = it % kStages;
            mbar_wait(&sm.k_full[s], (it / kStages) & 1);
            tc_fence_after();
            const uint32_t b = (sp_base_it + i) & 1;
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const uint64_t da = make_desc_sw128(smem_u32(sm.q[h]) + k * 32, 16, 1024);
                const uint64_t db = make_desc_sw128(smem_u32(sm.k[s][h]) + k * 32, 16, 1024);
                mma_ss(t_s[b], da, db, idesc_qk, (h | k) ? 1u : 0u);
              }
            mma_commit(&sm.s_full[b]);
            if (i == n - 1) mma_commit(&sm.q_empty);
          }
          if (i >= 1) {
            const int j = i - 1;
            const uint32_t it = kv_base_it + j;
            const int s = it % kStages;
            const uint32_t spj = sp_base_it + j;
            const uint32_t b = spj & 1;
            mbar_wait(&sm.p_full[b], (spj >> 1) & 1);
            mbar_wait(&sm.v_full[s], (it / kStages) & 1);
            if (j == 0) mbar_wait(&sm.o_empty, (item_it & 1) ^ 1);
            tc_fence_after();
            // keys of this tile that any row may see, rounded up to the MMA K step
            const int kt = W.kt_begin + j;
            int valid = kt < T.n_pref_tiles ? min(kBN, T.kv_len_max - kt * kBN)
                                            : min(kBN, T.lk1 - T.lk0 - (kt - T.n_pref_tiles) * kBN);
            const int ksteps = (valid + 15) >> 4;
            for (int k = 0; k < ksteps; ++k) {
              const uint64_t db = make_desc_sw128(smem_u32(sm.v[s][0]) + k * 2048, kHalfBytes, 1024);
              mma_ts(t_o, t_s[b] + k * 8, db, idesc_pv, (j | k) ? 1u : 0u);
            }
            mma_commit(&sm.kv_empty[s]);
            mma_commit(&sm.pv_done);
          }
        }
        kv_it += n; sp_it += n;
      }
    }
  } else {
    // ===================== softmax + epilogue: one thread per stacked row =====================
    const int quad = warp & 3;                         // TMEM lane group this warp may access
    const int r = quad * 32 + lane;                    // row of the tile
    const uint32_t lane_addr = (uint32_t)(quad * 32) << 16;
    uint32_t sp_it = 0, pv_it = 0;
    for (int w = blockIdx.x; w < n_work; w += gridDim.x) {
      const WorkRec W = p.plan.work[w];
      const TileRec T = p.plan.tiles[W.tile];
      const int n = W.kt_end - W.kt_begin;
      // ---- this row's token, head and lane ----
      const int tok_local = r / p.n_rep;
      const int head = W.g * p.n_rep + (r - tok_local * p.n_rep);
      const int tok = T.q_tok0 + tok_local;
      bool valid = tok_local < T.n_tok;
      int prefix_len = 0, ls = 0, le = 0;
      if (valid) {
        valid = false;
        for (int l = T.lane_first; l < T.lane_first + T.lane_count; ++l) {
          const int qs = p.lanes[l].q_start, ql = p.lanes[l].q_len;
          if (tok >= qs && tok < qs + ql) { prefix_len = p.lanes[l].prefix_len; ls = qs; le = qs + ql; valid = true; }
        }
      }
      float m_used = -INFINITY, l_sum = 0.f;           // m_used in raw score units

      for (int i = 0; i < n; ++i, ++sp_it) {
        const int kt = W.kt_begin + i;
        const uint32_t b = sp_it & 1;
        mbar_wait(&sm.s_full[b], (sp_it >> 1) & 1);
        tc_fence_after();
        float s[kBN];
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32_f(t_s[b] + lane_addr + c * 32, s + c * 32);
        tmem_wait_ld();
        // visible columns of this tile for this row: [lo, hi)
        int lo = 0, hi = 0;
        bool need_mask;
        if (kt < T.n_pref_tiles) {
          hi = min(kBN, prefix_len - kt * kBN);
          need_mask = (kt + 1) * kBN > T.kv_len_min || !valid;
        } else {
          const int base = T.lk0 + (kt - T.n_pref_tiles) * kBN;
          lo = max(0, ls - base); hi = min(kBN, le - base);
          need_mask = true;
        }
        if (!valid) { lo = 0; hi = 0; }
        if (need_mask) {
#pragma unroll
          for (int c = 0; c < kBN; ++c) s[c] = (c >= lo && c < hi) ? s[c] : -INFINITY;
        }
        float mx = s[0];
#pragma unroll
        for (int c = 1; c < kBN; ++c) mx = fmaxf(mx, s[c]);
        // PV of the previous key tile must have landed before O may be rescaled
        if (i > 0) { mbar_wait(&sm.pv_done, pv_it & 1); ++pv_it; tc_fence_after(); }
        const float m_new = fmaxf(m_used, mx);
        bool grow = false;
        if (m_used == -INFINITY) m_used = m_new;         // nothing accumulated yet (O row is 0 or unwritten)
        else grow = (m_new - m_used) * p.scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {             // warp-uniform: tcgen05.ld/st are .sync.aligned
          const float alpha = grow ? exp2f((m_used - m_new) * p.scale_log2) : 1.0f;
          if (grow) { l_sum *= alpha; m_used = m_new; }
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
        const float mb = (m_used == -INFINITY) ? 0.f : m_used * p.scale_log2;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int e = 0; e < 16; ++e) {
            const float p0 = exp2f(fmaf(s[c * 32 + 2 * e], p.scale_log2, -mb));
            const float p1 = exp2f(fmaf(s[c * 32 + 2 * e + 1], p.scale_log2, -mb));
            l_sum += p0 + p1;
            pk[e] = pack_bf16x2(p0, p1);
          }
          tmem_st16(t_s[b] + lane_addr + c * 16, pk);
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(&sm.p_full[b]);
      }
      // ---- epilogue ----
      mbar_wait(&sm.pv_done, pv_it & 1); ++pv_it;
      tc_fence_after();
      const float inv = l_sum > 0.f ? 1.0f / l_sum : 0.f;
      const float lse = l_sum > 0.f ? (m_used * p.scale_log2 + log2f(l_sum)) / kLog2e : -INFINITY;
      if (W.part_slot < 0) {
        __nv_bfloat16* orow = p.out + ((long long)tok * p.n_q_heads + head) * kD;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          float o[32];
          tmem_ld32_f(t_o + lane_addr + c * 32, o);
          tmem_wait_ld();
          if (valid) {
            uint32_t pk[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) pk[e] = pack_bf16x2(o[2 * e] * inv, o[2 * e + 1] * inv);
            uint4* dst = reinterpret_cast<uint4*>(orow + c * 32);
#pragma unroll
            for (int e = 0; e < 4; ++e) dst[e] = make_uint4(pk[4 * e], pk[4 * e + 1], pk[4 * e + 2], pk[4 * e + 3]);
          }
        }
        if (valid && p.lse) p.lse[(long long)tok * p.n_q_heads + head] = lse;
      } else {
        float* prow = p.plan.part_o + ((long long)W.part_slot * kBM + r) * kD;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          float o[32];
          tmem_ld32_f(t_o + lane_addr + c * 32, o);
          tmem_wait_ld();
          if (valid) {
            float4* dst = reinterpret_cast<float4*>(prow + c * 32);
#pragma unroll
            for (int e = 0; e < 8; ++e)
              dst[e] = make_float4(o[4 * e] * inv, o[4 * e + 1] * inv, o[4 * e + 2] * inv, o[4 * e + 3] * inv);
          }
        }
        if (valid) p.plan.part_lse[(long long)W.part_slot * kBM + r] = lse;
      }
      tc_fence_before();
      mbar_arrive(&sm.o_empty);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { __syncwarp(); tmem_dealloc<512>(tmem); }
}

// ---------------------------------------------------------------------------------------------
// combine: merge the split-KV partials of every split tile (one warp per stacked row)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
lane_combine_kernel(Plan plan, int n_q_heads, int n_kv_heads, int n_rep, __nv_bfloat16* __restrict__ out,
                    float* __restrict__ lse_out) {
  const int n_tiles = plan.hdr->n_tiles;
  const int t = blockIdx.x / n_kv_heads, g = blockIdx.x - t * n_kv_heads;
  if (t >= n_tiles) return;
  const TileRec T = plan.tiles[t];
  if (T.n_splits <= 1) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_rows = T.n_tok * n_rep;
  const int slot0 = T.part_base + g * T.n_splits;
  for (int r = warp; r < n_rows; r += 8) {
    float mx = -INFINITY;
    for (int s = 0; s < T.n_splits; ++s) mx = fmaxf(mx, plan.part_lse[(long long)(slot0 + s) * kBM + r]);
    float wsum = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < T.n_splits; ++s) {
      const float ls = plan.part_lse[(long long)(slot0 + s) * kBM + r];
      const float wgt = (ls == -INFINITY) ? 0.f : exp2f((ls - mx) * kLog2e);
      if (wgt > 0.f) {
        const float4 v = reinterpret_cast<const float4*>(plan.part_o + ((long long)(slot0 + s) * kBM + r) * kD)[lane];
        acc.x = fmaf(wgt, v.x, acc.x); acc.y = fmaf(wgt, v.y, acc.y);
        acc.z = fmaf(wgt, v.z, acc.z); acc.w = fmaf(wgt, v.w, acc.w);
      }
      wsum += wgt;
    }
    const float inv = 1.0f / wsum;
    const int tok_local = r / n_rep;
    const int head = g * n_rep + (r - tok_local * n_rep);
    const long long row = (long long)(T.q_tok0 + tok_local) * n_q_heads + head;
    uint2 pk;
    pk.x = pack_bf16x2(acc.x * inv, acc.y * inv);
    pk.y = pack_bf16x2(acc.z * inv, acc.w * inv);
    reinterpret_cast<uint2*>(out + row * kD)[lane] = pk;
    if (lse_out && lane == 0) lse_out[row] = mx + logf(wsum);
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
Bounds bounds_for(const al_attn_shape* s, int n_lanes, int total_q_rows, int n_sms) {
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  const int tpt = kBM / n_rep;
  Bounds b;
  b.max_tiles = ceil_div(total_q_rows, tpt) + n_lanes;
  b.max_work = b.max_tiles * s->n_kv_heads + n_sms;
  b.max_part = 2 * n_sms + 2 * s->n_kv_heads;
  return b;
}

struct WsLayout {
  size_t hdr, tiles, work, part_lse, part_o, total;
};
WsLayout ws_layout(const al_attn_shape* s, const Bounds& b) {
  WsLayout L;
  size_t off = 0;
  auto take = [&](size_t n) { size_t o = off; off = al_round_up(off + n, 256); return o; };
  L.hdr = take(sizeof(PlanHeader));
  L.tiles = take(sizeof(TileRec) * (size_t)b.max_tiles);
  L.work = take(sizeof(WorkRec) * (size_t)b.max_work);
  L.part_lse = take(sizeof(float) * (size_t)b.max_part * kBM);
  L.part_o = take(sizeof(float) * (size_t)b.max_part * kBM * kD);
  L.total = off;
  return L;
}

constexpr int kSmsForBounds = 160;   // workspace sizing when no handle is at hand (>= SMs of any B200)

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

}  // namespace

bool al_attention_umma_supported(const al_attn_shape* s) {
  if (s->dtype != AL_BF16 || s->head_dim != kD) return false;
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  return n_rep >= 1 && n_rep <= kBM;
}

size_t al_attention_umma_workspace_bytes(const al_handle* h, const al_attn_shape* s, int n_lanes, int total_q_rows,
                                         int max_prefix_len) {
  (void)max_prefix_len;
  const Bounds b = bounds_for(s, n_lanes, total_q_rows, h ? h->sm_count : kSmsForBounds);
  return ws_layout(s, b).total;
}

al_status al_launch_attention_umma(const al_handle* h, const al_attn_shape* s, float scale, const void* q,
                                   const void* k_new, const void* v_new, const void* k_cache, const void* v_cache,
                                   const al_lane_desc* lanes, int n_lanes, int total_q_rows, int max_prefix_len,
                                   void* out, float* lse, void* workspace, size_t workspace_bytes, cudaStream_t st) {
  (void)max_prefix_len;
  if (n_lanes > kMaxPlanLanes) AL_FAIL(AL_ERR_UNSUPPORTED, "al_lane_attention: more than %d lanes", kMaxPlanLanes);
  const int n_rep = s->n_q_heads / s->n_kv_heads;
  const int tpt = kBM / n_rep;
  // the workspace may have been sized without a handle (kSmsForBounds): use the bound it was sized for
  Bounds b = bounds_for(s, n_lanes, total_q_rows, h->sm_count);
  WsLayout L = ws_layout(s, b);
  if (workspace_bytes < L.total) AL_FAIL(AL_ERR_WORKSPACE, "al_lane_attention: workspace %zu < %zu", workspace_bytes, L.total);
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  Plan plan;
  plan.hdr = reinterpret_cast<PlanHeader*>(ws + L.hdr);
  plan.tiles = reinterpret_cast<TileRec*>(ws + L.tiles);
  plan.work = reinterpret_cast<WorkRec*>(ws + L.work);
  plan.part_lse = reinterpret_cast<float*>(ws + L.part_lse);
  plan.part_o = reinterpret_cast<float*>(ws + L.part_o);

  CUtensorMap mq, mkn, mvn, mkc, mvc;
  al_status rc;
  const uint64_t T = (uint64_t)total_q_rows, Hq = (uint64_t)s->n_q_heads, Hkv = (uint64_t)s->n_kv_heads;
  const uint64_t rowb = kD * 2;
  if ((rc = make_map_3d(h, &mq, q, kD, Hq, T, rowb, Hq * rowb, 64, (uint32_t)n_rep, (uint32_t)tpt)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mkn, k_new, kD, Hkv, T, rowb, Hkv * rowb, 64, 1, kBN)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mvn, v_new, kD, Hkv, T, rowb, Hkv * rowb, 64, 1, kBN)) != AL_OK) return rc;
  // a group with no prefix never touches the cache maps; encode them over k_new when there is no cache
  const uint64_t crows = s->cache_rows > 0 && k_cache ? (uint64_t)s->cache_rows : 1;
  const void* kc = (s->cache_rows > 0 && k_cache) ? k_cache : k_new;
  const void* vc = (s->cache_rows > 0 && v_cache) ? v_cache : v_new;
  if ((rc = make_map_3d(h, &mkc, kc, kD, crows, Hkv, rowb, crows * rowb, 64, kBN, 1)) != AL_OK) return rc;
  if ((rc = make_map_3d(h, &mvc, vc, kD, crows, Hkv, rowb, crows * rowb, 64, kBN, 1)) != AL_OK) return rc;

  lane_plan_kernel<<<1, 256, 0, st>>>(lanes, n_lanes, s->n_kv_heads, tpt, h->sm_count, b, plan);
  AL_CUDA_OK(cudaGetLastError());

  AttnParams p;
  p.lanes = lanes; p.plan = plan; p.out = static_cast<__nv_bfloat16*>(out); p.lse = lse;
  p.n_q_heads = s->n_q_heads; p.n_kv_heads = s->n_kv_heads; p.n_rep = n_rep;
  p.scale_log2 = scale * kLog2e;
  p.q_box_bytes = (uint32_t)(2 * tpt * n_rep * 64 * 2);
  const size_t smem = sizeof(AttnSmem) + 1024;
  AL_CUDA_OK(cudaFuncSetAttribute(lane_attention_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int grid = b.max_work < h->sm_count ? b.max_work : h->sm_count;
  lane_attention_umma_kernel<<<grid, kThreads, smem, st>>>(mq, mkn, mvn, mkc, mvc, p);
  AL_CUDA_OK(cudaGetLastError());
  lane_combine_kernel<<<b.max_tiles * s->n_kv_heads, 256, 0, st>>>(plan, s->n_q_heads, s->n_kv_heads, n_rep,
                                                                    static_cast<__nv_bfloat16*>(out), lse);
  AL_CUDA_OK(cudaGetLastError());
  h->launches += 3;
  return AL_OK;
}
