// al_lm_head_confidence -- the LM head fused with the transfer rule (the step upstream of
// PAPER.md L78-80 / Eq.8): logits[i][v] = <hidden[i], weight[v]> are produced tile by tile on the tensor cores
// and consumed in the epilogue by the online (max, first argmax, sum exp) recurrence of al_confidence_select -- the
// [N][V] logits, 90 % of a step's bytes when they are materialised, never exist in HBM.
//
// K5  lm_head_kernel<BN>: persistent, warp-specialised, one CTA per SM.
//       warp 0      TMA producer: A = hidden tile [128 rows][64], B = weight tile [BN rows][64] per K step, through a
//                   ring of kStages stages (128-byte swizzle, K-major operands: both matrices are read as stored)
//       warp 1      MMA issuer (one elected lane): tcgen05.mma kind::f16, M = 128, N = BN, K = 16, SS form, into one of
//                   two TMEM accumulators; tcgen05.commit frees the stage / publishes the accumulator
//       warps 4-7   epilogue: one thread per row reads its BN fp32 logits from TMEM 32 columns at a time and folds them
//                   into the row's running (m, s, idx) -- registers, across ALL vocabulary tiles of the unit -- while
//                   the issuer fills the other accumulator
//     unit = (128-row tile, contiguous chunk of vocabulary tiles); units are numbered chunk-major so that the CTAs
//     running at the same time share weight tiles through L2; a unit leaves one (m, s, idx) per row in the workspace
//     and lm_head_select_kernel merges a row's chunks in vocabulary order (first maximiser wins) and applies the
//     commit rule.  BN = 128 for one row tile (the weight stream is HBM-bound and small tiles balance the SMs), 256 else.
//     One row tile, kCluster = 2: every CTA would re-read the same hidden tile for each of its vocabulary tiles (L2 -> SM
//     traffic twice the weight stream), so the two CTAs of a cluster take alternate vocabulary tiles of one unit and
//     each loads HALF of the hidden tile with TMA multicast into both; a stage is reused once BOTH issuers'
//     tcgen05.commit (multicast to both CTAs' barriers) have released it.
#include <cuda_bf16.h>

#include "al_internal.h"
#include "al_ptx.cuh"

using namespace alptx;

namespace {

constexpr int kBM = 128, kBK = 64;
constexpr int kThreads = 256;
constexpr float kLog2e = 1.4426950408889634f;
constexpr int kNoIdx = 0x7fffffff;

template <int BN> struct Cfg {
  static constexpr int kStages = BN == 256 ? 4 : 6;
  static constexpr int kABytes = kBM * kBK * 2, kBBytes = BN * kBK * 2;
};

template <int BN> struct LmSmem {
  alignas(1024) uint8_t a[Cfg<BN>::kStages][Cfg<BN>::kABytes];
  alignas(1024) uint8_t b[Cfg<BN>::kStages][Cfg<BN>::kBBytes];
  uint64_t full[Cfg<BN>::kStages], empty[Cfg<BN>::kStages];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};

struct LmParams {
  int n_rows, vocab, hidden_dim;
  int m_tiles, n_tiles, n_chunks;          // unit u = chunk * m_tiles + m_tile; chunk j = vocabulary tiles [j n_tiles / n_chunks, ...)
                                           // (cluster of 2: a unit is a PAIR of chunks 2j, 2j+1 taking alternate tiles of the pair's range)
  int eos_id, n_lanes;
  const al_lane_desc* lanes;
  float4* parts;                           // [n_chunks][m_tiles * 128]  (m, s, idx bits, unused)
};

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// The vocabulary tiles [t0, t0 + step * count) one CTA takes of unit u: the whole chunk (no cluster), or every
// kCluster-th tile of the group's range starting at its rank (the range is rounded up to a multiple of the cluster
// size -- tiles beyond it are masked in the epilogue -- so that all ranks run equally long).
template <int kCluster>
__device__ __forceinline__ void unit_tiles(const LmParams& p, int u, int rank, int& chunk, int& mt, int& t0, int& count, int& step,
                                           int& t_end) {
  const int group = u / p.m_tiles;                         // chunk (no cluster) or pair of chunks
  mt = u - group * p.m_tiles;
  if (kCluster == 1) {
    chunk = group;
    t0 = (int)((long long)group * p.n_tiles / p.n_chunks);
    t_end = (int)((long long)(group + 1) * p.n_tiles / p.n_chunks);
    count = t_end - t0;
    step = 1;
  } else {
    const int n_groups = p.n_chunks / kCluster;
    const int a = (int)((long long)group * p.n_tiles / n_groups), b = (int)((long long)(group + 1) * p.n_tiles / n_groups);
    chunk = kCluster * group + rank;
    t0 = a + rank;
    count = (b - a + kCluster - 1) / kCluster;
    step = kCluster;
    t_end = b;                                             // a rank's last tile may be the next unit's (range not a multiple of the cluster): masked
  }
}

template <int BN, int kCluster>
__global__ void __launch_bounds__(kThreads, 1)
lm_head_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b, const LmParams p) {
  using C = Cfg<BN>;
  const int rank = kCluster > 1 ? (int)cluster_ctarank() : 0;
  const int cta = kCluster > 1 ? (int)blockIdx.x / kCluster : (int)blockIdx.x;      // cluster (or CTA) index
  const int n_ctas = (int)gridDim.x / kCluster;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  LmSmem<BN>& sm = *reinterpret_cast<LmSmem<BN>*>(smem_raw);
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    if (smem_u32(smem_raw) & 1023u) __trap();
    for (int s = 0; s < C::kStages; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kCluster); }
    for (int a = 0; a < 2; ++a) { mbar_init(&sm.acc_full[a], 1); mbar_init(&sm.acc_empty[a], 128); }
    fence_barrier_init();
    prefetch_tensormap(&map_a); prefetch_tensormap(&map_b);
  }
  if (warp == 1) tmem_alloc<512>(&sm.tmem_base);
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  if (kCluster > 1) cluster_sync_all();                    // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  const int k_steps = (p.hidden_dim + kBK - 1) / kBK;
  const int n_units = p.m_tiles * (p.n_chunks / kCluster);

  if (warp == 0 && lane == 0) {
    // ===================== TMA producer =====================
    uint32_t it = 0;
    for (int u = cta; u < n_units; u += n_ctas) {
      int chunk, mt, t0, count, step, t_end;
      unit_tiles<kCluster>(p, u, rank, chunk, mt, t0, count, step, t_end);
      for (int j = 0; j < count; ++j)
        for (int kb = 0; kb < k_steps; ++kb, ++it) {
          const int s = it % C::kStages;
          mbar_wait_relaxed(&sm.empty[s], ((it / C::kStages) & 1) ^ 1);      // released by every CTA of the cluster
          mbar_arrive_expect_tx(&sm.full[s], C::kABytes + C::kBBytes);
          if (kCluster == 1) {
            tma_load_2d(sm.a[s], &map_a, &sm.full[s], kb * kBK, mt * kBM);
          } else {                                                           // my half of the hidden tile, into both CTAs
            tma_load_2d_multicast(sm.a[s] + rank * (C::kABytes / kCluster), &map_a, &sm.full[s], kb * kBK,
                                  mt * kBM + rank * (kBM / kCluster), (uint16_t)((1u << kCluster) - 1u));
          }
          tma_load_2d(sm.b[s], &map_b, &sm.full[s], kb * kBK, (t0 + j * step) * BN);
        }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (warp-uniform loop, one elected lane issues) =====================
    const bool leader = elect_one();
    const uint32_t idesc = make_idesc_bf16(kBM, BN, 0, 0);
    const uint64_t da0 = make_desc_sw128(smem_u32(sm.a[0]), 16, 1024);
    const uint64_t db0 = make_desc_sw128(smem_u32(sm.b[0]), 16, 1024);
    uint32_t it = 0, tile = 0;
    for (int u = cta; u < n_units; u += n_ctas) {
      int chunk, mt, t0, count, step, t_end;
      unit_tiles<kCluster>(p, u, rank, chunk, mt, t0, count, step, t_end);
      for (int j = 0; j < count; ++j, ++tile) {
        const uint32_t acc = tile & 1;
        mbar_wait(&sm.acc_empty[acc], ((tile >> 1) & 1) ^ 1);            // the epilogue has read this accumulator
        tc_fence_after();
        const uint32_t d = tmem + acc * 256;
        for (int kb = 0; kb < k_steps; ++kb, ++it) {
          const int s = it % C::kStages;
          mbar_wait(&sm.full[s], (it / C::kStages) & 1);
          tc_fence_after();
          const uint64_t da = da0 + (uint64_t)(s * (C::kABytes >> 4)), db = db0 + (uint64_t)(s * (C::kBBytes >> 4));
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k)
            if (leader) mma_ss(d, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), idesc, (kb | k) ? 1u : 0u);
          if (leader) {
            if (kCluster == 1) mma_commit(&sm.empty[s]);
            else mma_commit_multicast(&sm.empty[s], (uint16_t)((1u << kCluster) - 1u));   // the stage holds parts the peers loaded: all release it
          }
        }
        if (leader) mma_commit(&sm.acc_full[acc]);
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: one thread per row, running (m, s, idx) over the unit's vocabulary tiles ==========
    const int quad = warp & 3;
    const int r = quad * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(quad * 32) << 16;
    uint32_t tile = 0;
    for (int u = cta; u < n_units; u += n_ctas) {
      int chunk, mt, t0, count, step, t_end;
      unit_tiles<kCluster>(p, u, rank, chunk, mt, t0, count, step, t_end);
      const int row = mt * kBM + r;
      int sup = -1;                                        // EOS suppressed on rows of refine lanes
      if (p.eos_id >= 0 && p.lanes)
        for (int l = 0; l < p.n_lanes; ++l) {
          const int qs = p.lanes[l].q_start, ql = p.lanes[l].q_len;
          if ((p.lanes[l].flags & AL_LANE_FLAG_REFINE) && row >= qs && row < qs + ql) sup = p.eos_id;
        }
      float m = -INFINITY, s = 0.f;
      int idx = kNoIdx;
      for (int j = 0; j < count; ++j, ++tile) {
        const int nt = t0 + j * step;
        const uint32_t acc = tile & 1;
        mbar_wait(&sm.acc_full[acc], (tile >> 1) & 1);
        tc_fence_after();
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
          uint32_t raw[32];
          tmem_ld32(tmem + acc * 256 + lane_addr + c * 32, raw);
          tmem_wait_ld();
          const int v0 = nt * BN + c * 32;
          float x[32];
#pragma unroll
          for (int e = 0; e < 32; ++e) {
            const int v = v0 + e;
            x[e] = (v < p.vocab && v != sup && nt < t_end) ? __uint_as_float(raw[e]) : -INFINITY;   // vocabulary tail, EOS, padding tile
          }
          float cm = x[0];
#pragma unroll
          for (int e = 1; e < 32; ++e) cm = fmaxf(cm, x[e]);
          if (cm > m) {                                    // strict >: earlier columns keep ties (first maximiser)
            s *= ex2f((m - cm) * kLog2e);                  // m = -inf: s is 0 and stays 0
            m = cm;
            int first = 31;
#pragma unroll
            for (int e = 30; e >= 0; --e) first = (x[e] == cm) ? e : first;
            idx = v0 + first;
          }
          const float mb = (m == -INFINITY) ? 0.f : m * kLog2e;
          float s0 = 0.f, s1 = 0.f;
#pragma unroll
          for (int e = 0; e < 32; e += 2) {
            s0 += ex2f(fmaf(x[e], kLog2e, -mb));
            s1 += ex2f(fmaf(x[e + 1], kLog2e, -mb));
          }
          s += s0 + s1;
        }
        tc_fence_before();
        mbar_arrive(&sm.acc_empty[acc]);                   // the accumulator may be overwritten
      }
      p.parts[(long long)chunk * (p.m_tiles * kBM) + row] = make_float4(m, s, __int_as_float(idx), 0.f);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (kCluster > 1) cluster_sync_all();                    // no CTA leaves while its peer may still write into it
  if (warp == 1) { __syncwarp(); tmem_dealloc<512>(tmem); }
}

// Merges a row's chunks in vocabulary order (strict >: the first maximiser wins, reading C6) and applies the commit
// rule of al_confidence_select.  One thread per row.
__global__ void __launch_bounds__(256)
lm_head_select_kernel(const float4* __restrict__ parts, int n_chunks, int rows_padded, int n_rows,
                      const int32_t* __restrict__ tokens_in, int mask_id, float threshold, float* __restrict__ conf_out,
                      int32_t* __restrict__ argmax_out, uint8_t* __restrict__ commit_out, int32_t* __restrict__ tokens_out) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int row = blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= n_rows) return;
  float m = -INFINITY, s = 0.f;
  int idx = kNoIdx;
  for (int j = 0; j < n_chunks; ++j) {
    const float4 q = parts[(long long)j * rows_padded + row];
    const int qi = __float_as_int(q.z);
    if (q.x > m) {
      s = s * ex2f((m - q.x) * kLog2e) + q.y;
      m = q.x; idx = qi;
    } else if (q.x > -INFINITY) {
      s += q.y * ex2f((q.x - m) * kLog2e);
      if (q.x == m && qi < idx) idx = qi;                 // the chunks of a cluster pair interleave: lowest index wins
    }
  }
  const float conf = 1.0f / s;
  const int tok = tokens_in[row];
  const bool commit = (tok == mask_id) && (conf >= threshold);
  conf_out[row] = conf;
  argmax_out[row] = idx;
  commit_out[row] = commit ? 1 : 0;
  tokens_out[row] = commit ? idx : tok;
}

struct LmPlan {
  int bn, cluster, m_tiles, n_tiles, n_chunks;
  size_t ws_bytes;
};
LmPlan lm_plan(int n_rows, int vocab, int sm_count) {
  LmPlan L;
  L.m_tiles = (n_rows + kBM - 1) / kBM;
  // one row tile (<= 128 rows): the weight stream is HBM-bound and what matters is equal bytes per SM -> small
  // vocabulary tiles, and the hidden tile shared by the two CTAs of a cluster (TMA multicast).  From two row tiles on
  // the wide tile wins (measured, 256 / 384 / 512 rows: 259 / 330 / 423 us against 293 / 407 / 528 us with 128-wide
  // tiles in clusters of 2, 283 / 373 / 500 us without clusters): half as many hidden-tile reads per weight byte.
  L.bn = L.m_tiles <= 1 ? 128 : 256;
  L.cluster = L.m_tiles <= 1 ? 2 : 1;
  L.n_tiles = (vocab + L.bn - 1) / L.bn;
  const int slots = sm_count / L.cluster;                  // CTAs, or clusters, that run at the same time
  // groups (chunks, or pairs of chunks): units = groups * m_tiles should fill whole waves of the slots (a last wave of
  // a few units would leave the others idle for a whole unit) while a CTA keeps at least 4 vocabulary tiles per unit;
  // the coarsest plan within 2 % of the best fill wins (fewer partials, longer register-resident runs)
  const int max_groups = L.n_tiles >= 4 * L.cluster ? L.n_tiles / (4 * L.cluster) : 1;
  auto fill_of = [&](int g) {
    const long long units = (long long)g * L.m_tiles;
    const long long waves = (units + slots - 1) / slots;
    return (double)units / (double)(waves * slots);
  };
  double best = 0.0;
  for (int g = 1; g <= max_groups; ++g) best = fill_of(g) > best ? fill_of(g) : best;
  long long groups = 1;
  for (int g = 1; g <= max_groups; ++g)
    if (fill_of(g) >= best - 0.02) { groups = g; break; }
  L.n_chunks = (int)groups * L.cluster;
  L.ws_bytes = (size_t)L.n_chunks * L.m_tiles * kBM * sizeof(float4);
  return L;
}

template <int BN, int kCluster>
al_status launch_lm_head(const al_handle* h, const CUtensorMap& ma, const CUtensorMap& mb, const LmParams& p, int n_units,
                         cudaStream_t cs) {
  const size_t smem = sizeof(LmSmem<BN>);
  AL_CUDA_OK(cudaFuncSetAttribute(lm_head_kernel<BN, kCluster>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int slots = h->sm_count / kCluster;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)((n_units < slots ? n_units : slots) * kCluster));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = cs;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = kCluster;
  attr[1].val.clusterDim.y = 1;
  attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = kCluster > 1 ? 2 : 1;
  AL_CUDA_OK(cudaLaunchKernelEx(&cfg, lm_head_kernel<BN, kCluster>, ma, mb, p));
  return AL_OK;
}

}  // namespace

al_status al_make_map_2d(const al_handle* h, CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols,
                         uint32_t box_rows);                 // al_selftest.cu
al_status al_launch_force_top1(al_handle* h, const al_lane_desc* lanes, int n_lanes, int n_rows, int mask_id,
                               const float* conf, const int32_t* argmax, uint8_t* commit, int32_t* tokens_out,
                               cudaStream_t cs);             // al_confidence.cu

extern "C" size_t al_lm_head_confidence_workspace_bytes(int32_t n_rows, int32_t vocab) {
  if (n_rows <= 0 || vocab <= 0) return 0;
  size_t worst = 0;
  for (int sms = 64; sms <= 256; sms += 4) {                 // (the handle is not at hand: bound over plausible SM counts)
    const size_t b = lm_plan(n_rows, vocab, sms).ws_bytes;
    worst = b > worst ? b : worst;
  }
  return al_round_up(worst, 256);
}

extern "C" al_status al_lm_head_confidence(al_handle* h, const void* hidden, const void* weight, int32_t n_rows,
                                           int32_t vocab, int32_t hidden_dim, const int32_t* tokens_in, int32_t mask_id,
                                           int32_t eos_id, float threshold, const al_lane_desc* lanes, int32_t n_lanes,
                                           int32_t flags, float* conf_out, int32_t* argmax_out, uint8_t* commit_out,
                                           int32_t* tokens_out, void* workspace, size_t workspace_bytes, void* stream) {
  const char* who = "al_lm_head_confidence";
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  if (n_rows < 0 || vocab < 0 || hidden_dim < 0 || n_lanes < 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: negative size", who);
  if (flags & ~AL_SELECT_FORCE_TOP1) AL_FAIL(AL_ERR_INVALID_ARG, "%s: unknown flags %d", who, flags);
  if (n_rows == 0) return AL_OK;
  al_status st = al_check_device(h, who);
  if (st != AL_OK) return st;
  if (vocab == 0 || hidden_dim == 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: vocab or hidden_dim is 0", who);
  if (hidden_dim % 8 != 0) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: hidden_dim %d must be a multiple of 8 (16-byte rows)", who, hidden_dim);
  if (!hidden || !weight || !tokens_in || !conf_out || !argmax_out || !commit_out || !tokens_out)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL pointer", who);
  if (!al_aligned16(hidden) || !al_aligned16(weight)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: hidden / weight must be 16-byte aligned", who);
  if (n_lanes > 0 && !lanes) AL_FAIL(AL_ERR_INVALID_ARG, "%s: n_lanes > 0 but lanes is NULL", who);
  if (eos_id >= vocab) AL_FAIL(AL_ERR_INVALID_ARG, "%s: eos_id %d >= vocab %d", who, eos_id, vocab);
  const LmPlan L = lm_plan(n_rows, vocab, h->sm_count);
  if (!workspace || !al_aligned16(workspace) || workspace_bytes < L.ws_bytes)
    AL_FAIL(AL_ERR_WORKSPACE, "%s: workspace %zu < %zu (or unaligned)", who, workspace_bytes, L.ws_bytes);
  CUtensorMap ma, mb;
  // (a cluster of 2 loads the hidden tile as two 64-row halves, one per CTA, multicast to both)
  if ((st = al_make_map_2d(h, &ma, hidden, (uint64_t)n_rows, (uint64_t)hidden_dim, (uint32_t)(kBM / L.cluster))) != AL_OK) return st;
  if ((st = al_make_map_2d(h, &mb, weight, (uint64_t)vocab, (uint64_t)hidden_dim, (uint32_t)L.bn)) != AL_OK) return st;
  LmParams p;
  p.n_rows = n_rows; p.vocab = vocab; p.hidden_dim = hidden_dim;
  p.m_tiles = L.m_tiles; p.n_tiles = L.n_tiles; p.n_chunks = L.n_chunks;
  p.eos_id = eos_id; p.n_lanes = n_lanes; p.lanes = n_lanes > 0 ? lanes : nullptr;
  p.parts = static_cast<float4*>(workspace);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  const int n_units = L.m_tiles * (L.n_chunks / L.cluster);
  st = L.cluster == 2 ? launch_lm_head<128, 2>(h, ma, mb, p, n_units, cs) : launch_lm_head<256, 1>(h, ma, mb, p, n_units, cs);
  if (st != AL_OK) return st;
  h->launches++;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)((n_rows + 255) / 256));
  cfg.blockDim = dim3(256);
  cfg.stream = cs;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  AL_CUDA_OK(cudaLaunchKernelEx(&cfg, lm_head_select_kernel, (const float4*)p.parts, L.n_chunks, L.m_tiles * kBM,
                                (int)n_rows, tokens_in, (int)mask_id, threshold, conf_out, argmax_out, commit_out,
                                tokens_out));
  h->launches++;
  if (flags & AL_SELECT_FORCE_TOP1)
    return al_launch_force_top1(h, n_lanes > 0 ? lanes : nullptr, n_lanes > 0 ? n_lanes : 1, n_rows, mask_id, conf_out,
                                argmax_out, commit_out, tokens_out, cs);
  return AL_OK;
}

// ---------------------------------------------------------------------------------------------
// al_lm_head_confidence_static: the same call for callers that cannot allocate (CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc): the per-(row, chunk) partials live in a file-scope device array
// instead of a caller-provided workspace.  Every GPU that loads the library holds the array until exit.
// ---------------------------------------------------------------------------------------------
namespace {
constexpr size_t kStaticScratchBytes = (size_t)AL_LM_HEAD_STATIC_SCRATCH_BYTES;   // 1 MiB = 65536 (m, s, idx) slots
static __device__ __align__(256) unsigned char g_lm_head_scratch[kStaticScratchBytes];
// In host code `g_lm_head_scratch` is a host-side stand-in, NOT a device address: the address a kernel may use comes
// from cudaGetSymbolAddress, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
void* g_scratch_ptr[kMaxDevices];               // zero-initialised; written once per device (same value from any thread)
}  // namespace

extern "C" size_t al_lm_head_confidence_static_max_bytes(void) { return kStaticScratchBytes; }

extern "C" al_status al_lm_head_confidence_static(al_handle* h, const void* hidden, const void* weight, int32_t n_rows,
                                                  int32_t vocab, int32_t hidden_dim, const int32_t* tokens_in,
                                                  int32_t mask_id, int32_t eos_id, float threshold,
                                                  const al_lane_desc* lanes, int32_t n_lanes, int32_t flags,
                                                  float* conf_out, int32_t* argmax_out, uint8_t* commit_out,
                                                  int32_t* tokens_out, void* stream) {
  const char* who = "al_lm_head_confidence_static";
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  if (n_rows < 0 || vocab < 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: negative size", who);
  if (n_rows == 0) return AL_OK;
  al_status st = al_check_device(h, who);       // the handle's device is the current one from here on
  if (st != AL_OK) return st;
  if (vocab == 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: vocab is 0", who);
  const size_t need = lm_plan(n_rows, vocab, h->sm_count).ws_bytes;
  if (need > kStaticScratchBytes)
    AL_FAIL(AL_ERR_UNSUPPORTED, "%s: %d rows x %d vocabulary entries need %zu bytes of scratch, the static array holds %zu "
            "(use al_lm_head_confidence with a workspace)", who, n_rows, vocab, need, kStaticScratchBytes);
  if (h->device < 0 || h->device >= kMaxDevices) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: device %d", who, h->device);
  void* ptr = g_scratch_ptr[h->device];
  if (!ptr) {
    AL_CUDA_OK(cudaGetSymbolAddress(&ptr, g_lm_head_scratch));
    g_scratch_ptr[h->device] = ptr;
  }
  // Nothing in the array has to start at zero: every slot the select kernel reads is written by this call's units.
  return al_lm_head_confidence(h, hidden, weight, n_rows, vocab, hidden_dim, tokens_in, mask_id, eos_id, threshold, lanes,
                               n_lanes, flags, conf_out, argmax_out, commit_out, tokens_out, ptr, kStaticScratchBytes, stream);
}
