// Host-side internals shared by the translation units of libasynclane (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "asynclane.h"

struct al_handle {
  int device;
  int sm_count;
  int cc_major, cc_minor;
  size_t smem_optin;
  mutable std::atomic<uint64_t> launches{0};   // kernels enqueued through this handle
  bool conf_spread = true; // confidence launches below one wave cap the CTAs per SM at the even share (ASYNCLANE_CONF_SPREAD=0 at al_create: off)
  bool self_plan = true;   // small attention calls plan inside the attention kernel (ASYNCLANE_SELF_PLAN=0 at al_create: always the plan kernel)
  // cuTensorMapEncodeTiled resolved through the runtime (no -lcuda at link time)
  CUresult (*encode_tiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                           const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                           CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                           CUtensorMapFloatOOBfill);
};

void al_set_error(const char* fmt, ...);

#define AL_FAIL(code, ...)     \
  do {                         \
    al_set_error(__VA_ARGS__); \
    return (code);             \
  } while (0)

#define AL_CUDA_OK(expr)                                                                   \
  do {                                                                                     \
    cudaError_t _e = (expr);                                                               \
    if (_e != cudaSuccess) AL_FAIL(AL_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
  } while (0)

static inline bool al_aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t al_round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int al_esize(int dtype) { return dtype == AL_BF16 ? 2 : 4; }

al_status al_check_shape(const al_attn_shape* s, const char* who);
al_status al_check_device(const al_handle* h, const char* who);

// ---- kernel launchers (each defined next to its kernels) ----------------------------------------
al_status al_launch_attention_simt(const al_handle* h, const al_attn_shape* s, float scale,
                                   const void* q, const void* k_new, const void* v_new,
                                   const void* k_cache, const void* v_cache,
                                   const al_lane_desc* lanes, int n_lanes, int total_q_rows,
                                   void* out, float* lse, cudaStream_t st);

size_t al_attention_umma_workspace_bytes(const al_handle* h_or_null, const al_attn_shape* s,
                                         int n_lanes, int total_q_rows, int max_prefix_len);
al_status al_launch_attention_umma(const al_handle* h, const al_attn_shape* s, float scale,
                                   const void* q, const void* k_new, const void* v_new,
                                   const void* k_cache, const void* v_cache,
                                   const al_lane_desc* lanes, int n_lanes, int total_q_rows,
                                   int max_prefix_len, void* out, float* lse, void* workspace,
                                   size_t workspace_bytes, cudaStream_t st);
al_status al_launch_plan_umma(const al_handle* h, const al_attn_shape* s, const al_lane_desc* lanes,
                              int n_lanes, int total_q_rows, int max_prefix_len, void* workspace,
                              size_t workspace_bytes, cudaStream_t st);
bool al_attention_umma_supported(const al_attn_shape* s);
// limits of the tensor-core path's plan (lanes, query tiles); AL_OK when the call fits
al_status al_attention_umma_check(const al_handle* h, const al_attn_shape* s, int n_lanes, int total_q_rows);

// ---- argument checks of the hot calls, shared with al_lane_step_host (nothing is enqueued) -------
al_status al_lane_attention_impl(int mode, const char* who, al_handle* h, const al_attn_shape* s, const void* q,
                                 const void* k_new, const void* v_new, const void* k_cache, const void* v_cache,
                                 const al_lane_desc* lanes, int32_t n_lanes, int32_t total_q_rows,
                                 int32_t max_prefix_len, void* out, float* lse, void* workspace,
                                 size_t workspace_bytes, void* stream);
al_status al_kv_refresh_check(const char* who, const al_handle* h, const al_attn_shape* s, const void* k_cache,
                              const void* v_cache, const void* k_src, const void* v_src, const int32_t* pos_dev,
                              int32_t n_pos, int32_t kv_base_row, int32_t n_layers, int64_t layer_stride_cache,
                              int64_t layer_stride_src);
al_status al_confidence_select_check(const char* who, const al_handle* h, const void* logits, int32_t dtype,
                                     int32_t n_rows, int32_t vocab, int64_t row_stride, const int32_t* tokens_in,
                                     int32_t eos_id, const al_lane_desc* lanes, int32_t n_lanes, int32_t flags,
                                     const float* conf_out, const int32_t* argmax_out, const uint8_t* commit_out,
                                     const int32_t* tokens_out);
