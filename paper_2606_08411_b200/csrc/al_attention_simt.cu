// K1c lane_attention (plain ALUs) -- the general path of al_lane_attention: fp32 I/O of any head_dim
// (BASELINE configs[0]) and bf16 shapes the tcgen05 kernel does not cover.  Same definition as the
// tensor-core kernel (Eq.2-3): row i of lane l attends to cache rows
// [kv_base_row, +prefix_len) of its kv-head and to the lane's own q_len new rows; nothing else.
//
// One CTA per packed token row, one warp per q-head (looping).  Keys are taken 32 at a time: lane j
// scores key j (q row staged in shared memory), the warp does the online-softmax update with
// shuffles, then every lane accumulates its head_dim/32 output columns over the 32 keys
// (coalesced V reads).  fp32 everywhere; exp2 with log2e folded into the scale.
#include <cuda_bf16.h>

#include "al_internal.h"

namespace {

constexpr int kWarps = 4;
constexpr int kMaxDPerLane = 8;   // head_dim <= 256
constexpr float kLog2e = 1.4426950408889634f;

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

template <typename T>
__global__ void __launch_bounds__(kWarps * 32)
lane_attention_simt_kernel(const T* __restrict__ q, const T* __restrict__ k_new, const T* __restrict__ v_new,
                           const T* __restrict__ k_cache, const T* __restrict__ v_cache,
                           const al_lane_desc* __restrict__ lanes, int n_lanes, int n_q_heads,
                           int n_kv_heads, int d, long long cache_rows, float scale_log2,
                           T* __restrict__ out, float* __restrict__ lse) {
  extern __shared__ float q_smem[];                      // [kWarps][d]
  __shared__ int s_lane;
  const int row = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) s_lane = -1;
  __syncthreads();
  for (int l = threadIdx.x; l < n_lanes; l += blockDim.x)
    if (row >= lanes[l].q_start && row < lanes[l].q_start + lanes[l].q_len) s_lane = l;
  __syncthreads();
  if (s_lane < 0) return;                                // row not covered by any lane: not written
  const al_lane_desc L = lanes[s_lane];
  const int n_rep = n_q_heads / n_kv_heads;
  const int n_keys = L.prefix_len + L.q_len;
  float* qs = q_smem + warp * d;
  const int dpl = (d + 31) / 32;

  for (int h = warp; h < n_q_heads; h += kWarps) {
    const int g = h / n_rep;
    const T* qrow = q + ((long long)row * n_q_heads + h) * d;
    __syncwarp();
    for (int c = lane; c < d; c += 32) qs[c] = to_f32(qrow[c]) * scale_log2;   // scores in log2 units
    __syncwarp();
    float m = -INFINITY, lsum = 0.f;
    float acc[kMaxDPerLane];
#pragma unroll
    for (int i = 0; i < kMaxDPerLane; ++i) acc[i] = 0.f;

    for (int j0 = 0; j0 < n_keys; j0 += 32) {
      const int j = j0 + lane;
      float s = -INFINITY;
      if (j < n_keys) {
        const T* kj = (j < L.prefix_len)
                          ? k_cache + ((long long)g * cache_rows + L.kv_base_row + j) * d
                          : k_new + ((long long)(L.q_start + j - L.prefix_len) * n_kv_heads + g) * d;
        float a = 0.f;
        for (int c = 0; c < d; ++c) a = fmaf(qs[c], to_f32(kj[c]), a);
        s = a;
      }
      float bm = s;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) bm = fmaxf(bm, __shfl_xor_sync(0xffffffffu, bm, off));
      const float m_new = fmaxf(m, bm);                  // finite: every batch has >= 1 valid key
      const float corr = exp2f(m - m_new);               // m = -inf on the first batch -> 0
      const float p = exp2f(s - m_new);                  // invalid keys: exp2(-inf) = 0
      float bs = p;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) bs += __shfl_xor_sync(0xffffffffu, bs, off);
      lsum = lsum * corr + bs;
      m = m_new;
#pragma unroll
      for (int i = 0; i < kMaxDPerLane; ++i) acc[i] *= corr;
      const int nb = min(32, n_keys - j0);
      for (int jj = 0; jj < nb; ++jj) {
        const float pj = __shfl_sync(0xffffffffu, p, jj);
        const int jk = j0 + jj;
        const T* vj = (jk < L.prefix_len)
                          ? v_cache + ((long long)g * cache_rows + L.kv_base_row + jk) * d
                          : v_new + ((long long)(L.q_start + jk - L.prefix_len) * n_kv_heads + g) * d;
#pragma unroll
        for (int i = 0; i < kMaxDPerLane; ++i)
          if (i < dpl) {
            const int c = i * 32 + lane;
            if (c < d) acc[i] = fmaf(pj, to_f32(vj[c]), acc[i]);
          }
      }
    }
    const float inv = 1.0f / lsum;
    T* orow = out + ((long long)row * n_q_heads + h) * d;
#pragma unroll
    for (int i = 0; i < kMaxDPerLane; ++i)
      if (i < dpl) {
        const int c = i * 32 + lane;
        if (c < d) orow[c] = from_f32<T>(acc[i] * inv);
      }
    if (lse && lane == 0) lse[(long long)row * n_q_heads + h] = (m + log2f(lsum)) / kLog2e;
  }
}

}  // namespace

al_status al_launch_attention_simt(const al_handle* h, const al_attn_shape* s, float scale,
                                   const void* q, const void* k_new, const void* v_new,
                                   const void* k_cache, const void* v_cache,
                                   const al_lane_desc* lanes, int n_lanes, int total_q_rows,
                                   void* out, float* lse, cudaStream_t st) {
  h->launches++;
  const size_t smem = (size_t)kWarps * s->head_dim * sizeof(float);
  const float scale_log2 = scale * kLog2e;
  if (s->dtype == AL_F32) {
    lane_attention_simt_kernel<float><<<total_q_rows, kWarps * 32, smem, st>>>(
        (const float*)q, (const float*)k_new, (const float*)v_new, (const float*)k_cache,
        (const float*)v_cache, lanes, n_lanes, s->n_q_heads, s->n_kv_heads, s->head_dim,
        (long long)s->cache_rows, scale_log2, (float*)out, lse);
  } else {
    lane_attention_simt_kernel<__nv_bfloat16><<<total_q_rows, kWarps * 32, smem, st>>>(
        (const __nv_bfloat16*)q, (const __nv_bfloat16*)k_new, (const __nv_bfloat16*)v_new,
        (const __nv_bfloat16*)k_cache, (const __nv_bfloat16*)v_cache, lanes, n_lanes, s->n_q_heads,
        s->n_kv_heads, s->head_dim, (long long)s->cache_rows, scale_log2, (__nv_bfloat16*)out, lse);
  }
  AL_CUDA_OK(cudaGetLastError());
  return AL_OK;
}
