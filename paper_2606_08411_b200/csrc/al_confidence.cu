// al_confidence_select -- per-position vocab softmax confidence / argmax / threshold unmask select
// (q_i and x^_i of Eq.8).
//
// K3  confidence_select_kernel: ONE launch, HBM-bound stream over logits [N][V].
//     A thread-block CLUSTER of k CTAs (k in {1,2,4,8}, chosen on the host so that N*k CTAs fill the
//     148 SMs) owns one row; CTA c streams the c-th contiguous chunk of the row.  A warp folds 2 KB
//     items (4 x 16-byte streaming loads per lane; two items in registers, the loads of the next one
//     issued before the current one is reduced) in two register passes:
//       pass A  packed bf16x2 max over the lane's 32 values -> warp max through one REDUX
//       pass B  sum += ex2(x*log2e - m*log2e): unpack, then per PAIR of elements one packed FFMA2, two
//               MUFU.EX2 and one packed FADD2 -- and for two pairs of every eight a degree-4 polynomial on
//               the FMA pipes instead of the MUFU (exp2_poly_pair).  At the HBM rate one ex2 per element
//               keeps the SM's 16-per-clock MUFU 75 % busy and the issue slots 70 %: the stream is bound by
//               all three at once, which is why instructions per element were counted (full items load
//               unpredicated, the EOS test is one warp-uniform compare per item).
//     keeping a warp-uniform running max m (rescaling the sum only when an item raises it) and the
//     first index attaining it.  Warps merge through shared memory, the CTAs of a cluster merge in
//     the leader's shared memory over DSMEM, and the leader applies the commit rule: no partials in
//     HBM, no second launch, no atomics.  Algorithmic bytes: N*V*esz (+ 17 N of tokens/outputs).
//     Merge op on (m, s, i): m' = max, s' = s1 e^{m1-m'} + s2 e^{m2-m'}, i' = index of the larger
//     m, lower index on ties -- associative, so the argmax is the first maximiser in any order.
// K3c force_top1: one warp per lane (optional flag, reading C4 of DESIGN.md).
#include <cooperative_groups.h>
#include <cuda_bf16.h>

#include "al_internal.h"

namespace cg = cooperative_groups;

namespace {

constexpr int kWarpVecs = 4;                 // 16-byte vectors per lane per item
constexpr int kItemVecs = 32 * kWarpVecs;    // 128 vectors = 2 KB per item; a warp keeps TWO items in registers
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxCluster = 8;
// Of every eight element pairs, those whose exponential runs on the FMA pipes (exp2_poly_pair) instead of the
// MUFU: one ex2 per element keeps the SM's 16-per-clock MUFU 75 % busy at the HBM rate, and below one wave of
// CTAs it is the busiest SM's MUFU, not HBM, that bounds the launch.
#ifndef AL_CONF_POLY_MASK
#define AL_CONF_POLY_MASK 0x88
#endif
constexpr uint32_t kPolyPairs = AL_CONF_POLY_MASK;
constexpr float kLog2e = 1.4426950408889634f;
constexpr int kNoIdx = 0x7fffffff;

struct Triple {
  float m;   // running max (natural units)
  float s;   // sum exp(x - m)
  int idx;   // first index attaining m
};

__device__ __forceinline__ int4 ld_stream(const void* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ float ex2(float x) {           // x <= 0 here (or -inf): flush-to-zero is exact enough
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
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
// 2^x for a pair on the FMA pipes, x <= 0 (or -inf): x = n + f, n = rint(x) read from the low mantissa bits of
// x + 1.5 * 2^23, f in [-0.5, 0.5]; 2^f by a degree-4 polynomial (relative error 2.7e-6 evaluated in fp32, mean
// 4e-8; the MUFU's ex2.approx is about 2e-7), 2^n by adding n to the exponent field.  Clamped at -126: padding
// and suppressed elements are -inf and contribute 2^-126 instead of 0, far below the rounding of a sum >= 1.
__device__ __forceinline__ void exp2_poly_pair(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  unpack2(x2, x0, x1);
  x2 = pack2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
  const uint64_t r2 = fadd2(x2, pack2(12582912.f, 12582912.f));
  const uint64_t f2 = ffma2(fadd2(r2, pack2(-12582912.f, -12582912.f)), pack2(-1.f, -1.f), x2);
  uint64_t q2 = ffma2(pack2(0.009570101276f, 0.009570101276f), f2, pack2(0.05591785908f, 0.05591785908f));
  q2 = ffma2(q2, f2, pack2(0.2402474433f, 0.2402474433f));
  q2 = ffma2(q2, f2, pack2(0.6931217909f, 0.6931217909f));
  q2 = ffma2(q2, f2, pack2(0.9999992847f, 0.9999992847f));
  float q0, q1, r0, r1;
  unpack2(q2, q0, q1);
  unpack2(r2, r0, r1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(r0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(r1) << 23));
}
// order-preserving float <-> int map, so that one integer REDUX gives the warp max of floats
__device__ __forceinline__ int f2ord(float f) {
  const int b = __float_as_int(f);
  return b ^ ((b >> 31) & 0x7fffffff);
}
__device__ __forceinline__ float ord2f(int o) { return __int_as_float(o ^ ((o >> 31) & 0x7fffffff)); }
__device__ __forceinline__ float warp_max(float v) { return ord2f(__reduce_max_sync(0xffffffffu, f2ord(v))); }

// (m, s, idx) (+)= (m2, s2, idx2); lower index wins ties so the result is order-independent.
__device__ __forceinline__ void combine(Triple& a, const Triple& b) {
  const bool take2 = (b.m > a.m) || (b.m == a.m && b.idx < a.idx);
  const float mn = fmaxf(a.m, b.m);
  const float ms = (mn == -INFINITY) ? 0.f : mn;          // all -inf so far: keep sums at 0
  a.s = a.s * ex2((a.m - ms) * kLog2e) + b.s * ex2((b.m - ms) * kLog2e);
  a.m = mn;
  a.idx = take2 ? b.idx : a.idx;
}

template <typename T> struct Vec;
template <> struct Vec<__nv_bfloat16> {
  static constexpr int kElems = 8;
  // max of the 8 values of one vector, folded into a packed bf16x2 running max
  __device__ static __forceinline__ void max_into(const int4& v, uint32_t& acc) {
    const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) asm("max.bf16x2 %0, %0, %1;" : "+r"(acc) : "r"(w[i]));
  }
  static constexpr uint32_t kAccInit = 0xff80ff80u;       // (-inf, -inf)
  __device__ static __forceinline__ float acc_max(uint32_t acc) {
    return fmaxf(__uint_as_float(acc << 16), __uint_as_float(acc & 0xffff0000u));
  }
  __device__ static __forceinline__ void unpack(const int4& v, float (&x)[8]) {
    const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      x[2 * i] = __uint_as_float(w[i] << 16);
      x[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
  __device__ static __forceinline__ void set_neg_inf(int4& v, int e) {
    const uint32_t sh = (e & 1) * 16, keep = ~(0xffffu << sh), ninf = 0xff80u << sh;   // static selects:
    const int w = e >> 1;                                    // no dynamic register indexing
    v.x = w == 0 ? (int)(((uint32_t)v.x & keep) | ninf) : v.x;
    v.y = w == 1 ? (int)(((uint32_t)v.y & keep) | ninf) : v.y;
    v.z = w == 2 ? (int)(((uint32_t)v.z & keep) | ninf) : v.z;
    v.w = w == 3 ? (int)(((uint32_t)v.w & keep) | ninf) : v.w;
  }
  __device__ static __forceinline__ float load1(const __nv_bfloat16* p) { return __bfloat162float(*p); }
};
template <> struct Vec<float> {
  static constexpr int kElems = 4;
  __device__ static __forceinline__ void max_into(const int4& v, uint32_t& acc) {
    float a = __uint_as_float(acc);
    a = fmaxf(fmaxf(a, __int_as_float(v.x)), fmaxf(__int_as_float(v.y), fmaxf(__int_as_float(v.z), __int_as_float(v.w))));
    acc = __float_as_uint(a);
  }
  static constexpr uint32_t kAccInit = 0xff800000u;       // -inf
  __device__ static __forceinline__ float acc_max(uint32_t acc) { return __uint_as_float(acc); }
  __device__ static __forceinline__ void unpack(const int4& v, float (&x)[4]) {
    x[0] = __int_as_float(v.x); x[1] = __int_as_float(v.y);
    x[2] = __int_as_float(v.z); x[3] = __int_as_float(v.w);
  }
  __device__ static __forceinline__ void set_neg_inf(int4& v, int e) {
    const int ninf = (int)0xff800000u;
    v.x = e == 0 ? ninf : v.x; v.y = e == 1 ? ninf : v.y;
    v.z = e == 2 ? ninf : v.z; v.w = e == 3 ? ninf : v.w;
  }
  __device__ static __forceinline__ float load1(const float* p) { return *p; }
};

// warp-cooperative: does `row` belong to a refine lane (EOS suppressed)?
__device__ __forceinline__ bool row_suppresses_eos(const al_lane_desc* lanes, int n_lanes, int row, int lane) {
  bool sup = false;
  for (int l = lane; l < n_lanes; l += 32) {
    const int qs = lanes[l].q_start, ql = lanes[l].q_len, fl = lanes[l].flags;
    sup |= (fl & AL_LANE_FLAG_REFINE) && row >= qs && row < qs + ql;
  }
  return __any_sync(0xffffffffu, sup);
}

// One element per lane (unaligned rows and the < 16-byte row tail): value x at vocabulary index e,
// or (-inf, kNoIdx) for idle lanes.  m and idx are warp-uniform, s is per lane.
__device__ __forceinline__ void fold_scalar(float x, int e, float& m, float& s, int& idx) {
  const float wm = warp_max(x);
  if (wm > m) {                                            // strict >: earlier items keep ties
    s *= ex2((m - wm) * kLog2e);                           // m = -inf: s is 0 and stays 0
    m = wm;
    idx = __reduce_min_sync(0xffffffffu, x == wm ? e : kNoIdx);
  }
  const float mb = (m == -INFINITY) ? 0.f : m * kLog2e;
  s += ex2(fmaf(x, kLog2e, -mb));
}

template <typename T>
__device__ __forceinline__ void load_item(int4 (&v)[kWarpVecs], const T* __restrict__ row, int vi0, int v_end) {
  const int4* src = reinterpret_cast<const int4*>(row) + vi0;
  if (vi0 - (int)(threadIdx.x & 31) + kItemVecs <= v_end) {          // warp-uniform: the whole item is in range
#pragma unroll
    for (int j = 0; j < kWarpVecs; ++j) v[j] = ld_stream(src + j * 32);
  } else {
    const int pad = (int)Vec<T>::kAccInit;
#pragma unroll
    for (int j = 0; j < kWarpVecs; ++j)
      v[j] = vi0 + j * 32 < v_end ? ld_stream(src + j * 32) : make_int4(pad, pad, pad, pad);
  }
}
// EOS suppression (refine rows only): element `sup` of the row becomes -inf in the item held in registers
template <typename T>
__device__ __forceinline__ void suppress_in_item(int4 (&v)[kWarpVecs], int vi0, int sup) {
  constexpr int E = Vec<T>::kElems;
  const int sv = sup / E;                                    // sup = -1: sv = 0 and the guard below fails
  if (sup >= 0 && (unsigned)(sv - (vi0 - (int)(threadIdx.x & 31))) < (unsigned)kItemVecs) {   // warp-uniform: this item holds it
#pragma unroll
    for (int j = 0; j < kWarpVecs; ++j)
      if (vi0 + j * 32 == sv) Vec<T>::set_neg_inf(v[j], sup - sv * E);
  }
}

// Fold one 4 KB item held in registers into the warp's running (m, idx) and the lane's sum s.
template <typename T>
__device__ __forceinline__ void fold_item(const int4 (&v)[kWarpVecs], int vi0, float& m, float& s, int& idx) {
  constexpr int E = Vec<T>::kElems;
  uint32_t acc = Vec<T>::kAccInit;
#pragma unroll
  for (int j = 0; j < kWarpVecs; ++j) Vec<T>::max_into(v[j], acc);
  const float lm = Vec<T>::acc_max(acc);
  const float wm = warp_max(lm);
  if (wm > m) {                                            // warp-uniform, rare after the first items
    s *= ex2((m - wm) * kLog2e);
    m = wm;
    int cand = kNoIdx;
    if (lm == wm) {
#pragma unroll
      for (int j = kWarpVecs - 1; j >= 0; --j) {           // descending, so the first maximiser wins
        float x[E];
        Vec<T>::unpack(v[j], x);
#pragma unroll
        for (int e = E - 1; e >= 0; --e)
          if (x[e] == wm) cand = (vi0 + j * 32) * E + e;
      }
    }
    idx = __reduce_min_sync(0xffffffffu, cand);
  }
  // packed fp32x2 FMA / ADD (sm_100): one issue slot per PAIR for the scaling and for the sum -- the stream is
  // bound by instruction issue before it is bound by HBM when fewer than four CTAs are resident per SM.  Each
  // half is the IEEE fma / add of the scalar form, the even elements in the low half, the odd ones in the high.
  const float mb = (m == -INFINITY) ? 0.f : m * kLog2e;
  const uint64_t l2 = pack2(kLog2e, kLog2e), nmb2 = pack2(-mb, -mb);
  uint64_t sum2 = pack2(0.f, 0.f);
#pragma unroll
  for (int j = 0; j < kWarpVecs; ++j) {
    float x[E];
    Vec<T>::unpack(v[j], x);
#pragma unroll
    for (int e = 0; e < E; e += 2) {
      const uint64_t t2 = ffma2(pack2(x[e], x[e + 1]), l2, nmb2);
      float a, b;
      if ((kPolyPairs >> ((j * (E / 2) + e / 2) & 7)) & 1u) {
        exp2_poly_pair(t2, a, b);
      } else {
        unpack2(t2, a, b);
        a = ex2(a); b = ex2(b);
      }
      sum2 = fadd2(sum2, pack2(a, b));
    }
  }
  float s0, s1;
  unpack2(sum2, s0, s1);
  s += s0 + s1;
}

struct SelectArgs {
  const int32_t* tokens_in;
  int mask_id;
  float threshold;
  float* conf_out;
  int32_t* argmax_out;
  uint8_t* commit_out;
  int32_t* tokens_out;
};

template <typename T, bool kVector>
__global__ void __launch_bounds__(kThreads, 4)
confidence_select_kernel(const T* __restrict__ logits, int n_rows, int vocab, long long row_stride, int k_cluster,
                         int eos_id, const al_lane_desc* __restrict__ lanes, int n_lanes, SelectArgs out) {
  constexpr int E = Vec<T>::kElems;
  __shared__ Triple s_warp[kWarps];
  __shared__ Triple s_cta[kMaxCluster];                    // leader CTA: one slot per cluster rank
  // programmatic dependent launch: overlaps the launch with the tail of the previous kernel in the
  // stream; everything that kernel wrote (the logits, in a real step) is visible after the wait
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int row = blockIdx.x / k_cluster;
  const int rank = blockIdx.x - row * k_cluster;
  const T* base = logits + (long long)row * row_stride;
  float m = -INFINITY, s = 0.f;
  int idx = kNoIdx;
  int sup = -1;
  // the row's token, read by the thread that applies the commit rule at the very end: in flight under the stream
  int tok = 0;
  if (threadIdx.x == 0 && rank == 0) tok = __ldg(out.tokens_in + row);

  if (kVector) {
    const int vec_total = vocab / E;
    const int vpc = (((vec_total + k_cluster - 1) / k_cluster) + 7) & ~7;   // vectors per chunk, 128-B aligned
    const int c0 = min(vec_total, rank * vpc), c1 = min(vec_total, c0 + vpc);
    // A warp keeps two 2 KB items in registers: the loads of item i + 1 are issued before item i is folded, so
    // that the memory system never waits for the arithmetic -- with all CTAs of a resident wave starting together
    // a load / fold / load loop runs the whole chip in lockstep (measured: 81 % of the copy bandwidth on one wave
    // of 592 rows against 97 % in steady state).  The first loads go out before anything else; whether the row
    // belongs to a refine lane (EOS suppressed) is looked up in the lane descriptors while they are in flight.
    constexpr int kStep = kWarps * kItemVecs;
    int i0 = c0 + warp * kItemVecs;
    int4 va[kWarpVecs], vb[kWarpVecs];
    if (i0 < c1) load_item<T>(va, base, i0 + lane, c1);
    if (i0 + kStep < c1) load_item<T>(vb, base, i0 + kStep + lane, c1);
    sup = (eos_id >= 0 && lanes && row_suppresses_eos(lanes, n_lanes, row, lane)) ? eos_id : -1;
    while (i0 < c1) {
      suppress_in_item<T>(va, i0 + lane, sup);
      fold_item<T>(va, i0 + lane, m, s, idx);
      if (i0 + 2 * kStep < c1) load_item<T>(va, base, i0 + 2 * kStep + lane, c1);
      i0 += kStep;
      if (i0 >= c1) break;
      suppress_in_item<T>(vb, i0 + lane, sup);
      fold_item<T>(vb, i0 + lane, m, s, idx);
      if (i0 + 2 * kStep < c1) load_item<T>(vb, base, i0 + 2 * kStep + lane, c1);
      i0 += kStep;
    }
    if (rank == k_cluster - 1 && warp == 0 && vec_total * E < vocab) {      // < 16-byte row tail
      const int e = vec_total * E + lane;
      const bool ok = e < vocab;
      fold_scalar(ok ? (e == sup ? -INFINITY : Vec<T>::load1(base + e)) : -INFINITY, ok ? e : kNoIdx, m, s, idx);
    }
  } else {                                                 // unaligned rows: one element per lane
    sup = (eos_id >= 0 && lanes && row_suppresses_eos(lanes, n_lanes, row, lane)) ? eos_id : -1;
    const int epc = (vocab + k_cluster - 1) / k_cluster;
    const int c0 = min(vocab, rank * epc), c1 = min(vocab, c0 + epc);
    for (int e0 = c0 + warp * 32; e0 < c1; e0 += kWarps * 32) {
      const int e = e0 + lane;
      const bool ok = e < c1;
      fold_scalar(ok ? (e == sup ? -INFINITY : Vec<T>::load1(base + e)) : -INFINITY, ok ? e : kNoIdx, m, s, idx);
    }
  }
  // lanes share m: the warp's sum is a plain add
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0) s_warp[warp] = Triple{m, s, idx};
  __syncthreads();
  Triple t{-INFINITY, 0.f, kNoIdx};
  if (warp == 0) {
    if (lane < kWarps) t = s_warp[lane];
#pragma unroll
    for (int off = kWarps / 2; off > 0; off >>= 1) {
      Triple o;
      o.m = __shfl_xor_sync(0xffffffffu, t.m, off);
      o.s = __shfl_xor_sync(0xffffffffu, t.s, off);
      o.idx = __shfl_xor_sync(0xffffffffu, t.idx, off);
      combine(t, o);
    }
  }
  if (k_cluster > 1) {
    cg::cluster_group cluster = cg::this_cluster();
    if (threadIdx.x == 0) cluster.map_shared_rank(s_cta, 0)[rank] = t;     // DSMEM store into the leader
    cluster.sync();
    if (rank != 0) return;
    if (warp == 0) {
      t = lane < k_cluster ? s_cta[lane] : Triple{-INFINITY, 0.f, kNoIdx};
#pragma unroll
      for (int off = kMaxCluster / 2; off > 0; off >>= 1) {
        Triple o;
        o.m = __shfl_xor_sync(0xffffffffu, t.m, off);
        o.s = __shfl_xor_sync(0xffffffffu, t.s, off);
        o.idx = __shfl_xor_sync(0xffffffffu, t.idx, off);
        combine(t, o);
      }
    }
  }
  if (threadIdx.x == 0) {
    const float conf = 1.0f / t.s;                         // = exp(max - logsumexp)
    const bool commit = (tok == out.mask_id) && (conf >= out.threshold);
    out.conf_out[row] = conf;
    out.argmax_out[row] = t.idx;
    out.commit_out[row] = commit ? 1 : 0;
    out.tokens_out[row] = commit ? t.idx : tok;
  }
}

// force-top1 (reading C4): one warp per lane; a lane with masked rows and no commit commits its
// masked row of largest confidence (lowest row on ties).  After the select kernel a still-masked
// row has tokens_out == mask_id and commit == 0.
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
  int best_row = kNoIdx;
  for (int i = lane; i < ql; i += 32) {
    const int row = qs + i;
    if (row < 0 || row >= n_rows) continue;
    const bool c = commit[row] != 0;
    any_commit |= c;
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
  if (lane == 0 && !any_commit && best_row != kNoIdx) {
    commit[best_row] = 1;
    tokens_out[best_row] = argmax[best_row];
  }
}

// cluster size: the largest k in {1,2,4,8} for which N*k CTAs still fit one resident wave
// (4 CTAs per SM) and every CTA keeps at least one 4 KB item per warp
int pick_cluster(int n_rows, int vec_total, int sm_count) {
  int k = 1;
  while (k < kMaxCluster && (long long)n_rows * (2 * k) <= 4LL * sm_count &&
         vec_total / (2 * k) >= 2 * kWarps * kItemVecs)
    k *= 2;
  return k;
}

constexpr int kSmemPerSm = 228 * 1024;      // shared memory of an sm_100 SM

template <typename T, bool kVector>
cudaError_t launch_select(int k, int n_rows, cudaStream_t cs, const T* logits, int vocab, long long row_stride,
                          int eos_id, const al_lane_desc* lanes, int n_lanes, const SelectArgs& out, int sm_count, bool spread) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)(n_rows * k));
  cfg.blockDim = dim3(kThreads);
  // A launch of less than one resident wave (4 CTAs per SM) is as slow as its busiest SM, and the block scheduler
  // does not spread such a grid evenly: at 384 one-row CTAs on 148 SMs some SMs get four and 384 rows take longer
  // than 444 (measured: 26.0 us against 22.8 at V = 131072).  Unused dynamic shared memory caps the CTAs an SM
  // can hold at the even share ceil(CTAs / SMs), which forces the spread.
  cfg.dynamicSmemBytes = 0;
  const long long n_ctas = (long long)n_rows * k;
  const int share = (int)((n_ctas + sm_count - 1) / sm_count);
  if (share < 4 && spread) {
    cfg.dynamicSmemBytes = (size_t)(kSmemPerSm / share - 2048) & ~(size_t)1023;   // (static shared memory + 1 KB per CTA reserved by the system)
    const cudaError_t e = cudaFuncSetAttribute(confidence_select_kernel<T, kVector>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)cfg.dynamicSmemBytes);
    if (e != cudaSuccess) return e;
  }
  cfg.stream = cs;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)k;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.wait in the kernel
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, confidence_select_kernel<T, kVector>, logits, n_rows, vocab, row_stride, k, eos_id,
                            lanes, n_lanes, out);
}

}  // namespace

// The cluster/DSMEM merge keeps every partial on chip: no HBM workspace is needed.  The entry point stays in
// the ABI (callers size their arenas through it) and returns 0; al_confidence_select accepts workspace == NULL.
al_status al_launch_force_top1(al_handle* h, const al_lane_desc* lanes, int n_lanes, int n_rows, int mask_id,
                               const float* conf, const int32_t* argmax, uint8_t* commit, int32_t* tokens_out,
                               cudaStream_t cs) {
  force_top1_kernel<<<(n_lanes + kWarps - 1) / kWarps, kThreads, 0, cs>>>(lanes, n_lanes, n_rows, mask_id, conf, argmax,
                                                                         commit, tokens_out);
  AL_CUDA_OK(cudaGetLastError());
  h->launches++;
  return AL_OK;
}

extern "C" size_t al_confidence_select_workspace_bytes(int32_t n_rows, int32_t vocab) {
  (void)n_rows; (void)vocab;
  return 0;
}

al_status al_confidence_select_check(const char* who, const al_handle* h, const void* logits, int32_t dtype,
                                     int32_t n_rows, int32_t vocab, int64_t row_stride, const int32_t* tokens_in,
                                     int32_t eos_id, const al_lane_desc* lanes, int32_t n_lanes, int32_t flags,
                                     const float* conf_out, const int32_t* argmax_out, const uint8_t* commit_out,
                                     const int32_t* tokens_out) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  if (dtype != AL_F32 && dtype != AL_BF16) AL_FAIL(AL_ERR_INVALID_ARG, "%s: bad dtype %d", who, dtype);
  if (n_rows < 0 || vocab < 0 || n_lanes < 0 || row_stride < vocab)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: bad sizes n_rows %d vocab %d row_stride %lld", who, n_rows, vocab, (long long)row_stride);
  if (flags & ~AL_SELECT_FORCE_TOP1) AL_FAIL(AL_ERR_INVALID_ARG, "%s: unknown flags %d", who, flags);
  if (n_rows == 0) return AL_OK;
  const al_status st = al_check_device(h, who);
  if (st != AL_OK) return st;
  if (vocab == 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: vocab is 0", who);
  if (!logits || !tokens_in || !conf_out || !argmax_out || !commit_out || !tokens_out)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL pointer", who);
  if (n_lanes > 0 && !lanes) AL_FAIL(AL_ERR_INVALID_ARG, "%s: n_lanes > 0 but lanes is NULL", who);
  if (eos_id >= vocab) AL_FAIL(AL_ERR_INVALID_ARG, "%s: eos_id %d >= vocab %d", who, eos_id, vocab);
  if ((long long)n_rows * kMaxCluster > 0x7fffffffLL) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: too many rows", who);
  return AL_OK;
}

extern "C" al_status al_confidence_select(al_handle* h, const void* logits, int32_t dtype, int32_t n_rows,
                                          int32_t vocab, int64_t row_stride, const int32_t* tokens_in,
                                          int32_t mask_id, int32_t eos_id, float threshold,
                                          const al_lane_desc* lanes, int32_t n_lanes, int32_t flags,
                                          float* conf_out, int32_t* argmax_out, uint8_t* commit_out,
                                          int32_t* tokens_out, void* workspace, size_t workspace_bytes,
                                          void* stream) {
  (void)workspace; (void)workspace_bytes;
  const al_status st = al_confidence_select_check("al_confidence_select", h, logits, dtype, n_rows, vocab, row_stride,
                                                  tokens_in, eos_id, lanes, n_lanes, flags, conf_out, argmax_out,
                                                  commit_out, tokens_out);
  if (st != AL_OK) return st;
  if (n_rows == 0) return AL_OK;
  const int esz = al_esize(dtype);
  const bool vec = al_aligned16(logits) && ((row_stride * esz) % 16 == 0);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  const al_lane_desc* lanes_eff = n_lanes > 0 ? lanes : nullptr;
  const SelectArgs out{tokens_in, mask_id, threshold, conf_out, argmax_out, commit_out, tokens_out};
  const int k = vec ? pick_cluster(n_rows, vocab / (16 / esz), h->sm_count) : pick_cluster(n_rows, vocab / 8, h->sm_count);

  cudaError_t e;
  if (dtype == AL_BF16) {
    const __nv_bfloat16* p = static_cast<const __nv_bfloat16*>(logits);
    e = vec ? launch_select<__nv_bfloat16, true>(k, n_rows, cs, p, vocab, row_stride, eos_id, lanes_eff, n_lanes, out, h->sm_count, h->conf_spread)
            : launch_select<__nv_bfloat16, false>(k, n_rows, cs, p, vocab, row_stride, eos_id, lanes_eff, n_lanes, out, h->sm_count, h->conf_spread);
  } else {
    const float* p = static_cast<const float*>(logits);
    e = vec ? launch_select<float, true>(k, n_rows, cs, p, vocab, row_stride, eos_id, lanes_eff, n_lanes, out, h->sm_count, h->conf_spread)
            : launch_select<float, false>(k, n_rows, cs, p, vocab, row_stride, eos_id, lanes_eff, n_lanes, out, h->sm_count, h->conf_spread);
  }
  if (e != cudaSuccess) AL_FAIL(AL_ERR_CUDA, "al_confidence_select: launch failed: %s", cudaGetErrorString(e));
  h->launches++;
  if (flags & AL_SELECT_FORCE_TOP1) {
    const int nl = lanes_eff ? n_lanes : 1;
    force_top1_kernel<<<(nl + kWarps - 1) / kWarps, kThreads, 0, cs>>>(lanes_eff, nl, n_rows, mask_id, conf_out,
                                                                      argmax_out, commit_out, tokens_out);
    AL_CUDA_OK(cudaGetLastError());
    h->launches++;
  }
  return AL_OK;
}
