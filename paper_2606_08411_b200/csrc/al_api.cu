// Handle life cycle, error reporting, descriptor validation and the attention dispatch of
// libasynclane (C ABI in include/asynclane.h).
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "al_internal.h"

static thread_local char g_err[512] = "";

void al_set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

extern "C" const char* al_last_error(void) { return g_err; }
extern "C" const char* al_version(void) { return "asynclane-b200 0.1 sm_100a"; }

extern "C" al_status al_create(al_handle** out, int device) {
  if (!out) AL_FAIL(AL_ERR_INVALID_ARG, "al_create: out_handle is NULL");
  *out = nullptr;
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n == 0)
    AL_FAIL(AL_ERR_CUDA, "al_create: no CUDA device (%s); there is no CPU fallback",
            e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
  if (device < 0 || device >= n) AL_FAIL(AL_ERR_INVALID_ARG, "al_create: device %d of %d", device, n);
  // nothing is allocated and the caller's current device is untouched until every query has succeeded
  cudaDeviceProp p;
  AL_CUDA_OK(cudaGetDeviceProperties(&p, device));
  if (p.major != 10)
    AL_FAIL(AL_ERR_UNSUPPORTED, "al_create: device is sm_%d%d; this library is built for sm_100a only", p.major,
            p.minor);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
    AL_FAIL(AL_ERR_CUDA, "al_create: cuTensorMapEncodeTiled not available");
  al_handle* h = new al_handle();
  h->device = device;
  h->sm_count = p.multiProcessorCount;
  h->cc_major = p.major;
  h->cc_minor = p.minor;
  h->smem_optin = p.sharedMemPerBlockOptin;
  h->encode_tiled = reinterpret_cast<decltype(h->encode_tiled)>(fn);
  const char* sp = getenv("ASYNCLANE_SELF_PLAN");   // "0": small attention calls use the plan kernel too (tests compare the two)
  h->self_plan = !(sp && sp[0] == '0');
  const char* cs = getenv("ASYNCLANE_CONF_SPREAD");
  h->conf_spread = !(cs && cs[0] == '0');
  *out = h;
  return AL_OK;
}

extern "C" al_status al_destroy(al_handle* h) {
  delete h;
  return AL_OK;
}

extern "C" int32_t al_sm_count(const al_handle* h) { return h ? h->sm_count : 0; }
extern "C" uint64_t al_launch_count(const al_handle* h) { return h ? h->launches.load() : 0; }

static al_status check_shape(const al_attn_shape* s, const char* who) {
  if (!s) AL_FAIL(AL_ERR_INVALID_ARG, "%s: shape is NULL", who);
  if (s->dtype != AL_F32 && s->dtype != AL_BF16) AL_FAIL(AL_ERR_INVALID_ARG, "%s: bad dtype %d", who, s->dtype);
  if (s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->n_q_heads % s->n_kv_heads != 0)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: heads %d/%d", who, s->n_q_heads, s->n_kv_heads);
  if (s->head_dim <= 0 || s->cache_rows < 0 || s->reserved != 0)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: head_dim %d cache_rows %lld reserved %d", who, s->head_dim,
            (long long)s->cache_rows, s->reserved);
  if (!(s->scale >= 0.f) || std::isinf(s->scale)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: scale %f", who, s->scale);
  return AL_OK;
}

al_status al_check_shape(const al_attn_shape* s, const char* who) { return check_shape(s, who); }

// The handle's tensor maps, SM count and grid sizes belong to h->device, while launches go to the calling
// thread's CURRENT device: a mismatch is refused instead of silently launching elsewhere.
al_status al_check_device(const al_handle* h, const char* who) {
  int cur = -1;
  AL_CUDA_OK(cudaGetDevice(&cur));
  if (cur != h->device)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: current CUDA device %d is not the handle's device %d (cudaSetDevice first)", who,
            cur, h->device);
  return AL_OK;
}

extern "C" size_t al_lane_attention_workspace_bytes(const al_attn_shape* s, int32_t n_lanes,
                                                    int32_t total_q_rows, int32_t max_prefix_len) {
  if (!s || n_lanes <= 0 || total_q_rows <= 0) return 0;
  if (!al_attention_umma_supported(s)) return 0;
  return al_attention_umma_workspace_bytes(nullptr, s, n_lanes, total_q_rows, max_prefix_len);
}

// mode bit 0: build the plan; bit 1: run the attention; bit 2: validate like a full call, launch nothing
al_status al_lane_attention_impl(int mode, const char* who, al_handle* h, const al_attn_shape* s, const void* q,
                                     const void* k_new, const void* v_new, const void* k_cache,
                                     const void* v_cache, const al_lane_desc* lanes, int32_t n_lanes,
                                     int32_t total_q_rows, int32_t max_prefix_len, void* out, float* lse,
                                     void* workspace, size_t workspace_bytes, void* stream) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  al_status st = check_shape(s, who);
  if (st != AL_OK) return st;
  if (n_lanes < 0 || total_q_rows < 0 || max_prefix_len < 0) AL_FAIL(AL_ERR_INVALID_ARG, "%s: negative size", who);
  if (n_lanes == 0 || total_q_rows == 0) return AL_OK;
  if ((st = al_check_device(h, who)) != AL_OK) return st;
  if (!lanes) AL_FAIL(AL_ERR_INVALID_ARG, "%s: lanes is NULL", who);
  if (max_prefix_len > s->cache_rows) AL_FAIL(AL_ERR_INVALID_ARG, "%s: max_prefix_len > cache_rows", who);
  if (s->head_dim > 256 || s->head_dim % 8 != 0)
    AL_FAIL(AL_ERR_UNSUPPORTED, "%s: head_dim %d (need multiple of 8, <= 256)", who, s->head_dim);
  if (!al_aligned16(workspace)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: workspace must be 16-byte aligned", who);
  if (mode & 6) {
    if (!q || !k_new || !v_new || !out) AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL pointer", who);
    if (max_prefix_len > 0 && (!k_cache || !v_cache)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL cache", who);
    if (!al_aligned16(q) || !al_aligned16(k_new) || !al_aligned16(v_new) || !al_aligned16(k_cache) ||
        !al_aligned16(v_cache) || !al_aligned16(out))
      AL_FAIL(AL_ERR_INVALID_ARG, "%s: pointers must be 16-byte aligned", who);
  }
  const float scale = s->scale > 0.f ? s->scale : 1.0f / sqrtf((float)s->head_dim);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  if (al_attention_umma_supported(s)) {
    const size_t need = al_attention_umma_workspace_bytes(h, s, n_lanes, total_q_rows, max_prefix_len);
    if (workspace_bytes < need || (need && !workspace))
      AL_FAIL(AL_ERR_WORKSPACE, "%s: workspace %zu < %zu", who, workspace_bytes, need);
    if ((st = al_attention_umma_check(h, s, n_lanes, total_q_rows)) != AL_OK) return st;
    if (mode & 1) {
      st = al_launch_plan_umma(h, s, lanes, n_lanes, total_q_rows, max_prefix_len, workspace, workspace_bytes, cs);
      if (st != AL_OK) return st;
    }
    if (mode & 2)
      return al_launch_attention_umma(h, s, scale, q, k_new, v_new, k_cache, v_cache, lanes, n_lanes,
                                      total_q_rows, max_prefix_len, out, lse, workspace, workspace_bytes, cs);
    return AL_OK;
  }
  if (mode & 2)
    return al_launch_attention_simt(h, s, scale, q, k_new, v_new, k_cache, v_cache, lanes, n_lanes,
                                    total_q_rows, out, lse, cs);
  return AL_OK;
}

extern "C" al_status al_lane_attention(al_handle* h, const al_attn_shape* s, const void* q,
                                       const void* k_new, const void* v_new, const void* k_cache,
                                       const void* v_cache, const al_lane_desc* lanes, int32_t n_lanes,
                                       int32_t total_q_rows, int32_t max_prefix_len, void* out,
                                       float* lse, void* workspace, size_t workspace_bytes,
                                       void* stream) {
  return al_lane_attention_impl(3, "al_lane_attention", h, s, q, k_new, v_new, k_cache, v_cache, lanes, n_lanes,
                             total_q_rows, max_prefix_len, out, lse, workspace, workspace_bytes, stream);
}

extern "C" al_status al_lane_plan(al_handle* h, const al_attn_shape* s, const al_lane_desc* lanes,
                                  int32_t n_lanes, int32_t total_q_rows, int32_t max_prefix_len,
                                  void* workspace, size_t workspace_bytes, void* stream) {
  return al_lane_attention_impl(1, "al_lane_plan", h, s, nullptr, nullptr, nullptr, nullptr, nullptr, lanes, n_lanes,
                             total_q_rows, max_prefix_len, nullptr, nullptr, workspace, workspace_bytes, stream);
}

extern "C" al_status al_lane_attention_planned(al_handle* h, const al_attn_shape* s, const void* q,
                                               const void* k_new, const void* v_new, const void* k_cache,
                                               const void* v_cache, const al_lane_desc* lanes,
                                               int32_t n_lanes, int32_t total_q_rows, int32_t max_prefix_len,
                                               void* out, float* lse, void* workspace,
                                               size_t workspace_bytes, void* stream) {
  return al_lane_attention_impl(2, "al_lane_attention_planned", h, s, q, k_new, v_new, k_cache, v_cache, lanes,
                             n_lanes, total_q_rows, max_prefix_len, out, lse, workspace, workspace_bytes, stream);
}

extern "C" al_status al_validate_lanes(al_handle* h, const al_attn_shape* s, const al_lane_desc* lanes,
                                       int32_t n_lanes, int32_t total_q_rows) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_lanes: handle is NULL");
  al_status st = check_shape(s, "al_validate_lanes");
  if (st != AL_OK) return st;
  if (n_lanes < 0 || total_q_rows < 0) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_lanes: negative size");
  if (n_lanes == 0) return AL_OK;
  if (!lanes) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_lanes: lanes is NULL");
  std::vector<al_lane_desc> L(n_lanes);
  AL_CUDA_OK(cudaMemcpy(L.data(), lanes, sizeof(al_lane_desc) * n_lanes, cudaMemcpyDeviceToHost));
  std::vector<uint8_t> covered(total_q_rows, 0);
  for (int i = 0; i < n_lanes; ++i) {
    const al_lane_desc& l = L[i];
    if (l.q_len < 1 || l.q_start < 0 || (int64_t)l.q_start + l.q_len > total_q_rows)
      AL_FAIL(AL_ERR_INVALID_ARG, "lane %d: rows [%d,+%d) outside [0,%d)", i, l.q_start, l.q_len, total_q_rows);
    if (l.prefix_len < 0 || l.kv_base_row < 0 || (int64_t)l.kv_base_row + l.prefix_len > s->cache_rows)
      AL_FAIL(AL_ERR_INVALID_ARG, "lane %d: cache rows [%d,+%d) outside [0,%lld)", i, l.kv_base_row,
              l.prefix_len, (long long)s->cache_rows);
    for (int r = l.q_start; r < l.q_start + l.q_len; ++r) {
      if (covered[r]) AL_FAIL(AL_ERR_INVALID_ARG, "lane %d overlaps another lane at row %d", i, r);
      covered[r] = 1;
    }
    for (int j = 0; j < n_lanes; ++j)
      if (L[j].group_id == l.group_id && L[j].kv_base_row != l.kv_base_row)
        AL_FAIL(AL_ERR_INVALID_ARG, "lanes %d and %d share group %d but not kv_base_row", i, j, l.group_id);
  }
  return AL_OK;
}

extern "C" al_status al_validate_refresh(al_handle* h, const al_attn_shape* s, const int32_t* pos_dev,
                                         int32_t n_pos, int32_t kv_base_row) {
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_refresh: handle is NULL");
  al_status st = check_shape(s, "al_validate_refresh");
  if (st != AL_OK) return st;
  if (n_pos < 0 || kv_base_row < 0) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_refresh: negative size");
  if (n_pos == 0) return AL_OK;
  if (!pos_dev) AL_FAIL(AL_ERR_INVALID_ARG, "al_validate_refresh: pos is NULL");
  std::vector<int32_t> P(n_pos);
  AL_CUDA_OK(cudaMemcpy(P.data(), pos_dev, sizeof(int32_t) * n_pos, cudaMemcpyDeviceToHost));
  for (int r = 0; r < n_pos; ++r) {
    if (P[r] < 0 || (int64_t)kv_base_row + P[r] >= s->cache_rows)
      AL_FAIL(AL_ERR_INVALID_ARG, "refresh position %d: cache row %lld outside [0,%lld)", r,
              (long long)kv_base_row + P[r], (long long)s->cache_rows);
    if (r > 0 && P[r] <= P[r - 1])
      AL_FAIL(AL_ERR_INVALID_ARG, "refresh positions %d and %d (%d, %d) are not strictly increasing: a duplicate "
              "makes the scatter order-dependent", r - 1, r, P[r - 1], P[r]);
  }
  return AL_OK;
}
