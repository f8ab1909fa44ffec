// al_kv_refresh -- compact cache refresh scatter (Eq.12).
//
// cache[layer][g][kv_base_row + pos[r]][:] = src[layer][r][g][:] for K and V, as a pure bit copy in
// 16-byte vectors.  HBM-bound stream: algorithmic bytes = 2 planes x (read + write) x R x H_kv x
// row_bytes x layers (+ 4R for pos).  Source reads are fully contiguous; destination writes are
// contiguous runs of row_bytes (256 B for d=128 bf16).  Each thread moves UNROLL vectors of K and
// of V with all loads issued before the stores (memory-level parallelism), streaming cache hints on
// the read side (source rows are read exactly once).
#include "al_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kUnroll = 4;

__device__ __forceinline__ int4 ld_stream(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// vecs_per_row = row_bytes/16; one "item" = one 16-byte vector of one (layer, r, g) row.
__global__ void __launch_bounds__(kThreads)
kv_refresh_kernel(int4* __restrict__ k_cache, int4* __restrict__ v_cache,
                  const int4* __restrict__ k_src, const int4* __restrict__ v_src,
                  const int32_t* __restrict__ pos, int n_pos, int kv_base_row, int n_kv_heads,
                  long long cache_rows, int vecs_per_row, long long layer_stride_cache_vecs,
                  long long layer_stride_src_vecs, long long items_per_layer, long long total_items) {
  // programmatic dependent launch: the launch overlaps the tail of the previous kernel in the stream
  // (the attention that still reads the cache rows this kernel overwrites); its memory operations are
  // complete and visible after the wait.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const long long stride = (long long)gridDim.x * kThreads;
  long long i0 = (long long)blockIdx.x * kThreads + threadIdx.x;
  for (; i0 < total_items; i0 += stride * kUnroll) {
    int4 kv[kUnroll], vv[kUnroll];
    long long dst[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const long long i = i0 + u * stride;
      dst[u] = -1;
      if (i < total_items) {
        const long long layer = i / items_per_layer;
        const long long rem = i - layer * items_per_layer;      // (r * H_kv + g) * vecs_per_row + c
        const int c = (int)(rem % vecs_per_row);
        const long long rg = rem / vecs_per_row;
        const int g = (int)(rg % n_kv_heads);
        const int r = (int)(rg / n_kv_heads);
        const long long s = layer * layer_stride_src_vecs + rem;
        kv[u] = ld_stream(k_src + s);
        vv[u] = ld_stream(v_src + s);
        const long long row = (long long)g * cache_rows + kv_base_row + __ldg(pos + r);
        dst[u] = layer * layer_stride_cache_vecs + row * vecs_per_row + c;
      }
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u)
      if (dst[u] >= 0) {
        k_cache[dst[u]] = kv[u];
        v_cache[dst[u]] = vv[u];
      }
  }
}

// K2b kv_append_kernel (al_refresh_forward): cache[g][kv_base_row + prefix_len + i][:] = src[q_start + i][g][:] for every
// lane, K and V, as 16-byte vectors.  blockIdx.y = lane; the blocks of a lane stride over its q_len * H_kv * vecs items.
__global__ void __launch_bounds__(kThreads)
kv_append_kernel(int4* __restrict__ k_cache, int4* __restrict__ v_cache, const int4* __restrict__ k_src,
                 const int4* __restrict__ v_src, const al_lane_desc* __restrict__ lanes, int n_kv_heads,
                 long long cache_rows, int vecs_per_row) {
  // programmatic dependent launch: behind the attention that still reads the cache rows written here
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const al_lane_desc L = lanes[blockIdx.y];
  const long long items = (long long)L.q_len * n_kv_heads * vecs_per_row;
  const long long dst_row0 = (long long)L.kv_base_row + L.prefix_len;
  for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < items; i += (long long)gridDim.x * kThreads) {
    const int c = (int)(i % vecs_per_row);
    const long long rg = i / vecs_per_row;
    const int g = (int)(rg % n_kv_heads);
    const long long r = rg / n_kv_heads;
    const long long s = ((long long)(L.q_start + r) * n_kv_heads + g) * vecs_per_row + c;
    const long long d = ((long long)g * cache_rows + dst_row0 + r) * vecs_per_row + c;
    k_cache[d] = ld_stream(k_src + s);
    v_cache[d] = ld_stream(v_src + s);
  }
}

}  // namespace

// al_refresh_forward: the refresh forward of Eq.12 -- the lane-batched attention
// of the given ranges over [their older prefix ; themselves] on the tcgen05 path, then their K/V rows written into the
// cache behind that prefix.  The attention reads the cache before the append writes it (stream order).
extern "C" al_status al_refresh_forward(al_handle* h, const al_attn_shape* s, const void* q, const void* k_new,
                                        const void* v_new, void* k_cache, void* v_cache, const al_lane_desc* lanes,
                                        int32_t n_lanes, int32_t total_q_rows, int32_t max_prefix_len, void* out,
                                        float* lse, void* workspace, size_t workspace_bytes, void* stream) {
  const char* who = "al_refresh_forward";
  al_status st = al_lane_attention_impl(4, who, h, s, q, k_new, v_new, k_cache, v_cache, lanes, n_lanes, total_q_rows,
                                        max_prefix_len, out, lse, workspace, workspace_bytes, stream);
  if (st != AL_OK) return st;
  if (n_lanes == 0 || total_q_rows == 0) return AL_OK;
  if (!k_cache || !v_cache || s->cache_rows <= 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: no cache to write", who);
  const long long row_bytes = (long long)s->head_dim * al_esize(s->dtype);
  if (row_bytes % 16 != 0) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: head_dim*esize = %lld not a multiple of 16", who, row_bytes);
  st = al_lane_attention_impl(3, who, h, s, q, k_new, v_new, k_cache, v_cache, lanes, n_lanes, total_q_rows, max_prefix_len,
                              out, lse, workspace, workspace_bytes, stream);
  if (st != AL_OK) return st;
  const int vpr = (int)(row_bytes / 16);
  long long bx = ((long long)total_q_rows * s->n_kv_heads * vpr + kThreads * 4 - 1) / (kThreads * 4);
  bx = bx < 1 ? 1 : (bx > 32 ? 32 : bx);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)bx, (unsigned)n_lanes);
  cfg.blockDim = dim3(kThreads);
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.wait in the kernel
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  AL_CUDA_OK(cudaLaunchKernelEx(&cfg, kv_append_kernel, (int4*)k_cache, (int4*)v_cache, (const int4*)k_new,
                                (const int4*)v_new, lanes, (int)s->n_kv_heads, (long long)s->cache_rows, vpr));
  h->launches++;
  return AL_OK;
}

al_status al_kv_refresh_check(const char* who, const al_handle* h, const al_attn_shape* s, const void* k_cache,
                              const void* v_cache, const void* k_src, const void* v_src, const int32_t* pos_dev,
                              int32_t n_pos, int32_t kv_base_row, int32_t n_layers, int64_t layer_stride_cache,
                              int64_t layer_stride_src) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  al_status st = al_check_shape(s, who);
  if (st != AL_OK) return st;
  if (n_pos < 0 || n_layers < 0 || kv_base_row < 0 || layer_stride_cache < 0 || layer_stride_src < 0)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: negative size", who);
  if (n_pos == 0 || n_layers == 0) return AL_OK;
  if ((st = al_check_device(h, who)) != AL_OK) return st;
  if (!k_cache || !v_cache || !k_src || !v_src || !pos_dev) AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL pointer", who);
  const int esz = al_esize(s->dtype);
  const long long row_bytes = (long long)s->head_dim * esz;
  if (row_bytes % 16 != 0) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: head_dim*esize = %lld not a multiple of 16", who, row_bytes);
  if (!al_aligned16(k_cache) || !al_aligned16(v_cache) || !al_aligned16(k_src) || !al_aligned16(v_src))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: pointers must be 16-byte aligned", who);
  if ((layer_stride_cache * esz) % 16 != 0 || (layer_stride_src * esz) % 16 != 0)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: layer strides must be multiples of 16 bytes", who);
  if (n_layers > 1 && (layer_stride_cache < (int64_t)s->n_kv_heads * s->cache_rows * s->head_dim ||
                       layer_stride_src < (int64_t)n_pos * s->n_kv_heads * s->head_dim))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: layer strides smaller than one layer", who);
  return AL_OK;
}

extern "C" al_status al_kv_refresh(al_handle* h, const al_attn_shape* s, void* k_cache, void* v_cache,
                                   const void* k_src, const void* v_src, const int32_t* pos_dev,
                                   int32_t n_pos, int32_t kv_base_row, int32_t n_layers,
                                   int64_t layer_stride_cache, int64_t layer_stride_src, void* stream) {
  const al_status st = al_kv_refresh_check("al_kv_refresh", h, s, k_cache, v_cache, k_src, v_src, pos_dev, n_pos,
                                           kv_base_row, n_layers, layer_stride_cache, layer_stride_src);
  if (st != AL_OK) return st;
  if (n_pos == 0 || n_layers == 0) return AL_OK;
  const int esz = al_esize(s->dtype);
  const long long row_bytes = (long long)s->head_dim * esz;
  const int vpr = (int)(row_bytes / 16);
  const long long items_per_layer = (long long)n_pos * s->n_kv_heads * vpr;
  const long long total = items_per_layer * n_layers;
  long long blocks = (total + (long long)kThreads * kUnroll - 1) / ((long long)kThreads * kUnroll);
  const long long cap = (long long)h->sm_count * 16;       // grid-stride beyond 16 CTAs per SM
  if (blocks > cap) blocks = cap;
  h->launches++;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)blocks);
  cfg.blockDim = dim3(kThreads);
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.wait in the kernel
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  AL_CUDA_OK(cudaLaunchKernelEx(&cfg, kv_refresh_kernel, (int4*)k_cache, (int4*)v_cache, (const int4*)k_src,
                                (const int4*)v_src, pos_dev, (int)n_pos, (int)kv_base_row, (int)s->n_kv_heads,
                                (long long)s->cache_rows, vpr, (long long)(layer_stride_cache * esz / 16),
                                (long long)(layer_stride_src * esz / 16), items_per_layer, total));
  return AL_OK;
}
