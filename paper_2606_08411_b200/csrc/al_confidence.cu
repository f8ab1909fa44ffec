// al_confidence_select -- per-position vocab softmax confidence / argmax / threshold unmask select
// (q_i and x^_i of Eq.8).
//
// K3  confidence_partial: HBM-bound stream over logits [N][V].  A work item is one CHUNK of one row
//     (256 16-byte vectors = 4 KB); each WARP owns whole items (grid-stride), issues its 8 128-bit
//     streaming loads per lane up front, folds them into a per-lane online (max, sum-exp, first
//     argmax), reduces across the warp with shuffles and writes one 16-byte partial.  No block-level
//     synchronisation, no shared memory.  Algorithmic bytes: N*V*esz (+ 14 N of outputs).
// K3b confidence_finalize: one warp per row merges the row's partials with the associative combine
//     (m, s, i): m' = max, s' = s1 e^{m1-m'} + s2 e^{m2-m'}, i' = index of the larger m (lower index
//     on ties) and applies the commit rule; K3c force_top1: one warp per lane (optional flag).
#include <cuda_bf16.h>

#include "al_internal.h"

namespace {

constexpr int kWarpVecs = 8;                 // 16-byte vectors per lane per item
constexpr int kItemVecs = 32 * kWarpVecs;    // 256 vectors = 4 KB per item
constexpr int kThreads = 256;
constexpr float kLog2e = 1.4426950408889634f;

struct __align__(16) Partial {
  float m;   // running max (natural units)
  float s;   // sum exp(x - m)
  int idx;   // first index attaining m
  int pad;
};

__device__ __forceinline__ int4 ld_stream(const void* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

template <typename T> struct VecTraits;
template <> struct VecTraits<__nv_bfloat16> {
  static constexpr int kElems = 8;
  __device__ static __forceinline__ void unpack(const int4& v, float (&x)[8]) {
    const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      x[2 * i] = __uint_as_float(w[i] << 16);
      x[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
  __device__ static __forceinline__ float load1(const __nv_bfloat16* p) { return __bfloat162float(*p); }
};
template <> struct VecTraits<float> {
  static constexpr int kElems = 4;
  __device__ static __forceinline__ void unpack(const int4& v, float (&x)[4]) {
    x[0] = __int_as_float(v.x); x[1] = __int_as_float(v.y);
    x[2] = __int_as_float(v.z); x[3] = __int_as_float(v.w);
  }
  __device__ static __forceinline__ float load1(const float* p) { return *p; }
};

// (m, s, idx) (+)= (m2, s2, idx2); lower index wins ties so the result is order-independent.
__device__ __forceinline__ void combine(float& m, float& s, int& idx, float m2, float s2, int idx2) {
  const bool take2 = (m2 > m) || (m2 == m && idx2 < idx);
  const float mn = fmaxf(m, m2);
  const float ms = (mn == -INFINITY) ? 0.f : mn;          // all -inf so far: keep sums at 0
  s = s * exp2f((m - ms) * kLog2e) + s2 * exp2f((m2 - ms) * kLog2e);
  m = mn;
  idx = take2 ? idx2 : idx;
}

// warp-cooperative: does `row` belong to a refine lane (EOS suppressed)?
__device__ __forceinline__ bool row_suppresses_eos(const al_lane_desc* lanes, int n_lanes, int row, int lane) {
  bool sup = false;
  for (int l = lane; l < n_lanes; l += 32) {
    const int qs = lanes[l].q_start, ql = lanes[l].q_len, fl = lanes[l].flags;
    sup |= (fl & AL_LANE_FLAG_REFINE) && row >= qs && row < qs + ql;
  }
  return __any_sync(0xffffffffu, sup);
}

// fold n values x[0..n) whose first element has vocabulary index `base` into (m, s, idx)
template <int N>
__device__ __forceinline__ void fold(float (&x)[N], int base, float& m, float& s, int& idx) {
  float vm = x[0];
  int vi = 0;
#pragma unroll
  for (int i = 1; i < N; ++i)
    if (x[i] > vm) { vm = x[i]; vi = i; }                 // strict >: first maximiser inside the vector
  if (vm > m) {                                           // strict >: earlier vectors keep ties
    s *= exp2f((m - vm) * kLog2e);                        // m = -inf: s is 0 and exp2(-inf) = 0
    m = vm;
    idx = base + vi;
  }
  const float mb = (m == -INFINITY) ? 0.f : m * kLog2e;
#pragma unroll
  for (int i = 0; i < N; ++i) s += exp2f(fmaf(x[i], kLog2e, -mb));
}

template <typename T, bool kVector>
__global__ void __launch_bounds__(kThreads)
confidence_partial_kernel(const T* __restrict__ logits, int n_rows, int vocab, long long row_stride,
                          int items_per_row, int eos_id, const al_lane_desc* __restrict__ lanes,
                          int n_lanes, Partial* __restrict__ partials) {
  constexpr int E = VecTraits<T>::kElems;
  const int lane = threadIdx.x & 31;
  const long long warp = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
  const long long n_warps = ((long long)gridDim.x * kThreads) >> 5;
  const long long n_items = (long long)n_rows * items_per_row;
  const int vec_total = vocab / E;                         // whole vectors per row (vector path)

  for (long long item = warp; item < n_items; item += n_warps) {
    const int row = (int)(item / items_per_row);
    const int chunk = (int)(item - (long long)row * items_per_row);
    const T* base = logits + (long long)row * row_stride;
    const int sup = (eos_id >= 0 && lanes && row_suppresses_eos(lanes, n_lanes, row, lane)) ? eos_id : -1;
    float m = -INFINITY, s = 0.f;
    int idx = 0x7fffffff;

    if (kVector) {
      const int v0 = chunk * kItemVecs + lane;
      int4 v[kWarpVecs];
#pragma unroll
      for (int j = 0; j < kWarpVecs; ++j) {
        const int vi = v0 + j * 32;
        if (vi < vec_total) v[j] = ld_stream(base + (long long)vi * E);
      }
#pragma unroll
      for (int j = 0; j < kWarpVecs; ++j) {
        const int vi = v0 + j * 32;
        if (vi < vec_total) {
          float x[E];
          VecTraits<T>::unpack(v[j], x);
          const int sup_local = sup - vi * E;              // sup = -1 => negative
          if (sup_local >= 0 && sup_local < E) {
#pragma unroll
            for (int i = 0; i < E; ++i) x[i] = (i == sup_local) ? -INFINITY : x[i];
          }
          fold<E>(x, vi * E, m, s, idx);
        }
      }
      // scalar tail of the row (vocab % E elements) rides with the last item
      if (chunk == items_per_row - 1) {
        const int e = vec_total * E + lane;
        if (e < vocab) {
          float x[1] = {e == sup ? -INFINITY : VecTraits<T>::load1(base + e)};
          fold<1>(x, e, m, s, idx);
        }
      }
    } else {                                               // unaligned rows: element-wise, same items
      const int e0 = chunk * kItemVecs * E;
      const int e1 = min(vocab, e0 + kItemVecs * E);
      for (int e = e0 + lane; e < e1; e += 32) {
        float x[1] = {e == sup ? -INFINITY : VecTraits<T>::load1(base + e)};
        fold<1>(x, e, m, s, idx);
      }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const float m2 = __shfl_xor_sync(0xffffffffu, m, off);
      const float s2 = __shfl_xor_sync(0xffffffffu, s, off);
      const int i2 = __shfl_xor_sync(0xffffffffu, idx, off);
      combine(m, s, idx, m2, s2, i2);
    }
    if (lane == 0) partials[item] = Partial{m, s, idx, 0};
  }
}

__global__ void __launch_bounds__(kThreads)
confidence_finalize_kernel(const Partial* __restrict__ partials, int n_rows, int items_per_row,
                           const int32_t* __restrict__ tokens_in, int mask_id, float threshold,
                           float* __restrict__ conf_out, int32_t* __restrict__ argmax_out,
                           uint8_t* __restrict__ commit_out, int32_t* __restrict__ tokens_out) {
  const int lane = threadIdx.x & 31;
  const int row = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  if (row >= n_rows) return;
  float m = -INFINITY, s = 0.f;
  int idx = 0x7fffffff;
  for (int c = lane; c < items_per_row; c += 32) {
    const Partial p = partials[(long long)row * items_per_row + c];
    combine(m, s, idx, p.m, p.s, p.idx);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float m2 = __shfl_xor_sync(0xffffffffu, m, off);
    const float s2 = __shfl_xor_sync(0xffffffffu, s, off);
    const int i2 = __shfl_xor_sync(0xffffffffu, idx, off);
    combine(m, s, idx, m2, s2, i2);
  }
  if (lane == 0) {
    const float conf = 1.0f / s;                           // = exp(max - logsumexp)
    const int tok = tokens_in[row];
    const bool commit = (tok == mask_id) && (conf >= threshold);
    conf_out[row] = conf;
    argmax_out[row] = idx;
    commit_out[row] = commit ? 1 : 0;
    tokens_out[row] = commit ? idx : tok;
  }
}

// force-top1 (reading C4): one warp per lane; a lane with masked rows and no commit commits its
// masked row of largest confidence (lowest row on ties).  tokens_mask[] = commit-independent copy
// of "row is masked", taken from tokens_out/commit state written by finalize.
__global__ void __launch_bounds__(kThreads)
force_top1_kernel(const al_lane_desc* __restrict__ lanes, int n_lanes, int n_rows, int mask_id,
                  const float* __restrict__ conf, const int32_t* __restrict__ argmax,
                  uint8_t* __restrict__ commit, int32_t* __restrict__ tokens_out) {
  const int lane = threadIdx.x & 31;
  const int l = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  if (l >= n_lanes) return;
  int qs = 0, ql = n_rows;
  if (lanes) { qs = lanes[l].q_start; ql = lanes[l].q_len; }
  bool any_commit = false;
  float best = -1.f;
  int best_row = 0x7fffffff;
  for (int i = lane; i < ql; i += 32) {
    const int row = qs + i;
    if (row < 0 || row >= n_rows) continue;
    const bool c = commit[row] != 0;
    any_commit |= c;
    // after finalize a still-masked row has tokens_out == mask_id and commit == 0
    if (!c && tokens_out[row] == mask_id) {
      const float q = conf[row];
      if (q > best || (q == best && row < best_row)) { best = q; best_row = row; }
    }
  }
  any_commit = __any_sync(0xffffffffu, any_commit);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float b2 = __shfl_xor_sync(0xffffffffu, best, off);
    const int r2 = __shfl_xor_sync(0xffffffffu, best_row, off);
    if (b2 > best || (b2 == best && r2 < best_row)) { best = b2; best_row = r2; }
  }
  if (lane == 0 && !any_commit && best_row != 0x7fffffff) {
    commit[best_row] = 1;
    tokens_out[best_row] = argmax[best_row];
  }
}

inline int items_per_row_for(int vocab, int esz) {
  const int elems_per_item = kItemVecs * (16 / esz);
  return (vocab + elems_per_item - 1) / elems_per_item;
}

}  // namespace

extern "C" size_t al_confidence_select_workspace_bytes(int32_t n_rows, int32_t vocab) {
  if (n_rows <= 0 || vocab <= 0) return 0;
  return (size_t)n_rows * items_per_row_for(vocab, 4) * sizeof(Partial);   // f32 has the most items
}

extern "C" al_status al_confidence_select(al_handle* h, const void* logits, int32_t dtype, int32_t n_rows,
                                          int32_t vocab, int64_t row_stride, const int32_t* tokens_in,
                                          int32_t mask_id, int32_t eos_id, float threshold,
                                          const al_lane_desc* lanes, int32_t n_lanes, int32_t flags,
                                          float* conf_out, int32_t* argmax_out, uint8_t* commit_out,
                                          int32_t* tokens_out, void* workspace, size_t workspace_bytes,
                                          void* stream) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: handle is NULL");
  if (dtype != AL_F32 && dtype != AL_BF16) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: bad dtype %d", dtype);
  if (n_rows < 0 || vocab < 0 || n_lanes < 0 || row_stride < vocab)
    AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: bad sizes n_rows %d vocab %d row_stride %lld", n_rows, vocab, (long long)row_stride);
  if (flags & ~AL_SELECT_FORCE_TOP1) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: unknown flags %d", flags);
  if (n_rows == 0) return AL_OK;
  if (vocab == 0) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: vocab is 0");
  if (!logits || !tokens_in || !conf_out || !argmax_out || !commit_out || !tokens_out)
    AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: NULL pointer");
  if (n_lanes > 0 && !lanes) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: n_lanes > 0 but lanes is NULL");
  if (eos_id >= vocab) AL_FAIL(AL_ERR_INVALID_ARG, "al_confidence_select: eos_id %d >= vocab %d", eos_id, vocab);
  const int esz = al_esize(dtype);
  const int ipr = items_per_row_for(vocab, esz);
  const size_t need = (size_t)n_rows * ipr * sizeof(Partial);
  if (!workspace || workspace_bytes < need || !al_aligned16(workspace))
    AL_FAIL(AL_ERR_WORKSPACE, "al_confidence_select: workspace %zu < %zu (or unaligned)", workspace_bytes, need);
  const bool vec = al_aligned16(logits) && ((row_stride * esz) % 16 == 0);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  Partial* parts = static_cast<Partial*>(workspace);
  const al_lane_desc* lanes_eff = n_lanes > 0 ? lanes : nullptr;

  const long long n_items = (long long)n_rows * ipr;
  const int warps_per_block = kThreads / 32;
  long long blocks = (n_items + warps_per_block - 1) / warps_per_block;
  const long long cap = (long long)h->sm_count * 8;        // 8 x 256 threads = 64 warps per SM
  if (blocks > cap) blocks = cap;
#define AL_LAUNCH_PARTIAL(T, V)                                                                     \
  confidence_partial_kernel<T, V><<<(unsigned)blocks, kThreads, 0, cs>>>(                           \
      static_cast<const T*>(logits), n_rows, vocab, (long long)row_stride, ipr, eos_id, lanes_eff,  \
      n_lanes, parts)
  if (dtype == AL_BF16) { if (vec) AL_LAUNCH_PARTIAL(__nv_bfloat16, true); else AL_LAUNCH_PARTIAL(__nv_bfloat16, false); }
  else                  { if (vec) AL_LAUNCH_PARTIAL(float, true);         else AL_LAUNCH_PARTIAL(float, false); }
#undef AL_LAUNCH_PARTIAL
  AL_CUDA_OK(cudaGetLastError());
  h->launches += 2;
  const int fin_blocks = (n_rows + warps_per_block - 1) / warps_per_block;
  confidence_finalize_kernel<<<fin_blocks, kThreads, 0, cs>>>(parts, n_rows, ipr, tokens_in, mask_id, threshold,
                                                               conf_out, argmax_out, commit_out, tokens_out);
  AL_CUDA_OK(cudaGetLastError());
  if (flags & AL_SELECT_FORCE_TOP1) {
    const int nl = lanes_eff ? n_lanes : 1;
    force_top1_kernel<<<(nl + warps_per_block - 1) / warps_per_block, kThreads, 0, cs>>>(
        lanes_eff, nl, n_rows, mask_id, conf_out, argmax_out, commit_out, tokens_out);
    AL_CUDA_OK(cudaGetLastError());
    h->launches++;
  }
  return AL_OK;
}
