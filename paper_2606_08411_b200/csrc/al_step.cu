// al_lane_step_host -- the whole lane-batched denoising step driven from HOST buffers: the
// end-to-end entry of the C ABI (bench.py's `e2e` leg).  Host code only: it lays the per-step inputs
// (every layer's Q/K_new/V_new and refresh rows, the logits) out in a caller-provided device arena,
// validates all three parts, then enqueues the copies, one plan + one attention launch per layer, the
// layer-batched refresh and the confidence/select call on one stream and copies the results back.
// No arithmetic of the method lives here.
#include <cstring>

#include "al_internal.h"

namespace {

struct ArenaLayout {
  size_t q, k_new, v_new, lanes, k_src, v_src, pos, logits, tokens_in;        // inputs
  size_t out, conf, argmax, commit, tokens_out;                              // results
  size_t ws_attn, ws_conf;                                                    // kernel workspaces
  size_t n_q, n_kvnew, n_lanes, n_src, n_pos, n_logits, n_tok, n_out, n_ws_attn, n_ws_conf;
  size_t total;
};

bool layout(const al_attn_shape* s, const al_host_step* p, ArenaLayout* L) {
  if (!s || !p || p->n_lanes < 0 || p->total_q_rows < 0 || p->n_pos < 0 || p->n_rows < 0 || p->vocab < 0 ||
      p->max_prefix_len < 0 || p->n_layers < 0 || s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->head_dim <= 0)
    return false;
  const size_t esz = (size_t)al_esize(s->dtype);
  const size_t T = (size_t)p->total_q_rows, d = (size_t)s->head_dim;
  const size_t layers = (size_t)(p->n_layers > 0 ? p->n_layers : 1);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = al_round_up(off + bytes, 256); return o; };
  L->n_q = layers * T * s->n_q_heads * d * esz;                 // every layer's rows, layer-major
  L->n_kvnew = layers * T * s->n_kv_heads * d * esz;
  L->n_lanes = (size_t)p->n_lanes * sizeof(al_lane_desc);
  L->n_src = layers * (size_t)p->n_pos * s->n_kv_heads * d * esz;
  L->n_pos = (size_t)p->n_pos * 4;
  L->n_logits = (size_t)p->n_rows * p->vocab * esz;
  L->n_tok = (size_t)p->n_rows * 4;
  L->n_out = L->n_q;
  L->n_ws_attn = al_lane_attention_workspace_bytes(s, p->n_lanes, p->total_q_rows, p->max_prefix_len);
  L->n_ws_conf = al_confidence_select_workspace_bytes(p->n_rows, p->vocab);
  L->q = take(L->n_q); L->k_new = take(L->n_kvnew); L->v_new = take(L->n_kvnew);
  L->lanes = take(L->n_lanes); L->k_src = take(L->n_src); L->v_src = take(L->n_src);
  L->pos = take(L->n_pos); L->logits = take(L->n_logits); L->tokens_in = take(L->n_tok);
  L->out = take(L->n_out); L->conf = take(L->n_tok); L->argmax = take(L->n_tok);
  L->commit = take((size_t)p->n_rows); L->tokens_out = take(L->n_tok);
  L->ws_attn = take(L->n_ws_attn); L->ws_conf = take(L->n_ws_conf);
  L->total = off;
  return true;
}

}  // namespace

extern "C" size_t al_lane_step_host_arena_bytes(const al_attn_shape* s, const al_host_step* p) {
  ArenaLayout L;
  return layout(s, p, &L) ? L.total : 0;
}

extern "C" void al_lane_step_host_traffic(const al_attn_shape* s, const al_host_step* p, uint64_t* h2d,
                                          uint64_t* d2h) {
  ArenaLayout L;
  uint64_t in = 0, outb = 0;
  if (layout(s, p, &L)) {
    in = L.n_q + 2 * L.n_kvnew + L.n_lanes + 2 * L.n_src + L.n_pos + L.n_logits + L.n_tok;
    outb = L.n_out + 3 * L.n_tok + (uint64_t)p->n_rows;
  }
  if (h2d) *h2d = in;
  if (d2h) *d2h = outb;
}

extern "C" al_status al_lane_step_host(al_handle* h, const al_attn_shape* s, const al_host_step* p,
                                       void* k_cache, void* v_cache, void* arena, size_t arena_bytes,
                                       void* stream) {
  const char* who = "al_lane_step_host";
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  al_status st = al_check_shape(s, who);
  if (st != AL_OK) return st;
  ArenaLayout L;
  if (!layout(s, p, &L)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: bad step sizes", who);
  if (!arena || arena_bytes < L.total || (reinterpret_cast<uintptr_t>(arena) & 255u))
    AL_FAIL(AL_ERR_WORKSPACE, "%s: arena %zu < %zu (or not 256-byte aligned)", who, arena_bytes, L.total);
  const int layers = p->n_layers > 0 ? p->n_layers : 1;
  const size_t esz = (size_t)al_esize(s->dtype);
  const bool attn = p->n_lanes > 0 && p->total_q_rows > 0, refresh = p->n_pos > 0, conf = p->n_rows > 0;
  if (attn && (!p->q || !p->k_new || !p->v_new || !p->lanes || !p->out))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL attention buffer", who);
  if (refresh && (!p->k_src || !p->v_src || !p->pos)) AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL refresh buffer", who);
  if (conf && (!p->logits || !p->tokens_in || !p->conf || !p->argmax || !p->commit || !p->tokens_out))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL confidence buffer", who);
  if (conf && p->n_lanes > 0 && !p->lanes) AL_FAIL(AL_ERR_INVALID_ARG, "%s: lanes is NULL", who);
  const int64_t one_layer_cache = (int64_t)s->n_kv_heads * s->cache_rows * s->head_dim;
  if (layers > 1 && p->cache_layer_stride < one_layer_cache)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: cache_layer_stride %lld smaller than one layer (%lld elements)", who,
            (long long)p->cache_layer_stride, (long long)one_layer_cache);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  uint8_t* a = static_cast<uint8_t*>(arena);
  const al_lane_desc* lanes_dev = reinterpret_cast<const al_lane_desc*>(a + L.lanes);
  const size_t q_layer = L.n_q / layers, kv_layer = L.n_kvnew / layers;
  const int64_t src_layer_stride = (int64_t)p->n_pos * s->n_kv_heads * s->head_dim;
  // ---- every part is validated before the first copy is enqueued: on error nothing has been launched ----
  if (attn) {
    st = al_lane_attention_impl(4, who, h, s, a + L.q, a + L.k_new, a + L.v_new, k_cache, v_cache, lanes_dev,
                                p->n_lanes, p->total_q_rows, p->max_prefix_len, a + L.out, nullptr, a + L.ws_attn,
                                L.n_ws_attn, stream);
    if (st != AL_OK) return st;
  }
  if (refresh) {
    st = al_kv_refresh_check(who, h, s, k_cache, v_cache, a + L.k_src, a + L.v_src,
                             reinterpret_cast<const int32_t*>(a + L.pos), p->n_pos, p->refresh_base_row, layers,
                             p->cache_layer_stride, src_layer_stride);
    if (st != AL_OK) return st;
  }
  if (conf) {
    if (p->select_flags & ~AL_SELECT_FORCE_TOP1) AL_FAIL(AL_ERR_INVALID_ARG, "%s: unknown select_flags", who);
    st = al_confidence_select_check(who, h, a + L.logits, s->dtype, p->n_rows, p->vocab, p->vocab,
                                    reinterpret_cast<const int32_t*>(a + L.tokens_in), p->eos_id, lanes_dev,
                                    p->n_lanes, p->select_flags, reinterpret_cast<float*>(a + L.conf),
                                    reinterpret_cast<int32_t*>(a + L.argmax), a + L.commit,
                                    reinterpret_cast<int32_t*>(a + L.tokens_out));
    if (st != AL_OK) return st;
  }
  auto up = [&](size_t off, const void* src, size_t n) -> cudaError_t {
    return n ? cudaMemcpyAsync(a + off, src, n, cudaMemcpyHostToDevice, cs) : cudaSuccess;
  };
  auto down = [&](void* dst, size_t off, size_t n) -> cudaError_t {
    return n ? cudaMemcpyAsync(dst, a + off, n, cudaMemcpyDeviceToHost, cs) : cudaSuccess;
  };
  if (attn || conf) AL_CUDA_OK(up(L.lanes, p->lanes, L.n_lanes));
  if (attn) {
    AL_CUDA_OK(up(L.q, p->q, L.n_q));
    AL_CUDA_OK(up(L.k_new, p->k_new, L.n_kvnew));
    AL_CUDA_OK(up(L.v_new, p->v_new, L.n_kvnew));
    // the lanes are those of one scheduler iteration: one plan, then one planned launch per layer
    st = al_lane_plan(h, s, lanes_dev, p->n_lanes, p->total_q_rows, p->max_prefix_len, a + L.ws_attn, L.n_ws_attn,
                      stream);
    if (st != AL_OK) return st;
    for (int l = 0; l < layers; ++l) {
      const size_t co = (size_t)l * (size_t)p->cache_layer_stride * esz;
      st = al_lane_attention_planned(h, s, a + L.q + l * q_layer, a + L.k_new + l * kv_layer,
                                     a + L.v_new + l * kv_layer, static_cast<uint8_t*>(k_cache) + co,
                                     static_cast<uint8_t*>(v_cache) + co, lanes_dev, p->n_lanes, p->total_q_rows,
                                     p->max_prefix_len, a + L.out + l * q_layer, nullptr, a + L.ws_attn, L.n_ws_attn,
                                     stream);
      if (st != AL_OK) return st;
    }
    AL_CUDA_OK(down(p->out, L.out, L.n_out));
  }
  if (refresh) {
    AL_CUDA_OK(up(L.k_src, p->k_src, L.n_src));
    AL_CUDA_OK(up(L.v_src, p->v_src, L.n_src));
    AL_CUDA_OK(up(L.pos, p->pos, L.n_pos));
    st = al_kv_refresh(h, s, k_cache, v_cache, a + L.k_src, a + L.v_src, reinterpret_cast<const int32_t*>(a + L.pos),
                       p->n_pos, p->refresh_base_row, layers, p->cache_layer_stride, src_layer_stride, stream);
    if (st != AL_OK) return st;
  }
  if (conf) {
    AL_CUDA_OK(up(L.logits, p->logits, L.n_logits));
    AL_CUDA_OK(up(L.tokens_in, p->tokens_in, L.n_tok));
    st = al_confidence_select(h, a + L.logits, s->dtype, p->n_rows, p->vocab, p->vocab,
                              reinterpret_cast<const int32_t*>(a + L.tokens_in), p->mask_id, p->eos_id,
                              p->threshold, lanes_dev, p->n_lanes, p->select_flags,
                              reinterpret_cast<float*>(a + L.conf), reinterpret_cast<int32_t*>(a + L.argmax),
                              a + L.commit, reinterpret_cast<int32_t*>(a + L.tokens_out), a + L.ws_conf, L.n_ws_conf,
                              stream);
    if (st != AL_OK) return st;
    AL_CUDA_OK(down(p->conf, L.conf, L.n_tok));
    AL_CUDA_OK(down(p->argmax, L.argmax, L.n_tok));
    AL_CUDA_OK(down(p->commit, L.commit, (size_t)p->n_rows));
    AL_CUDA_OK(down(p->tokens_out, L.tokens_out, L.n_tok));
  }
  return AL_OK;
}
