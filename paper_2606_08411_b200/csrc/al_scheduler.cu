// al_scheduler_run -- AsyncLane active-lane decoding (Algorithm 1) of one sequence: host control
// flow around the device calls of this library.  Per iteration: the active lanes A_t (Eq.10
// L121) become lane descriptors, ONE model call evaluates all of them (Eq.11), al_confidence_select applies the
// transfer rule, al_lane_status returns 32 bytes per lane, and the host applies the fork operator (Eq.6),
// completion, successor spawning / cascading termination (Eq.9) and the periodic compact refresh (Eq.12).
// COLLECTDFS (L125) reconstructs the output.  Readings C18-C21 are spelled out in include/asynclane.h.
//
// The model is a callback; al_stub_model_fn (a table-driven stand-in: there are no weights in this repository) is the
// only kernel defined here.  No arithmetic of the transfer rule lives in this file.
#include <algorithm>
#include <cstring>
#include <vector>

#include "al_internal.h"

namespace {

constexpr int kGen = 0, kRef = 1;
constexpr int kActive = 0, kCompleted = 1, kForked = 2;

// logits[row][v] = base[pos][v] + gain * (step + 1) * (v == target[pos])
__global__ void stub_model_kernel(const float* __restrict__ base, const int32_t* __restrict__ target, float gain, int vocab,
                                  const int32_t* __restrict__ row_pos, const int32_t* __restrict__ row_step, int n_rows,
                                  float* __restrict__ logits) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)n_rows * vocab) return;
  const int row = (int)(i / vocab), v = (int)(i - (long long)row * vocab);
  const int pos = row_pos[row];
  float x = base[(long long)pos * vocab + v];
  if (v == target[pos]) x += gain * ((float)row_step[row] + 1.0f);
  logits[i] = x;
}

struct DeviceBuffers {                       // everything the run allocates; freed by the destructor
  uint8_t* dev = nullptr;
  uint8_t* pinned = nullptr;
  ~DeviceBuffers() {
    if (dev) cudaFree(dev);
    if (pinned) cudaFreeHost(pinned);
  }
};

struct Layout {                              // one device arena and its pinned mirror for the per-iteration copies
  size_t lanes, tokens_in, row_pos, row_step, up_bytes;            // host -> device, contiguous
  size_t status, tokens_out, commit, down_bytes;                   // device -> host, contiguous (offsets from `down`)
  size_t down, logits, conf, argmax, delims, nofork, iota, ws_attn, total;
};

}  // namespace

extern "C" int al_stub_model_fn(void* user, const al_lane_desc* lanes_host, const int32_t* lane_steps_host, int32_t n_lanes,
                                int32_t n_rows, const int32_t* row_pos_dev, const int32_t* tokens_dev, float* logits_dev,
                                void* stream) {
  (void)lanes_host; (void)lane_steps_host; (void)n_lanes; (void)tokens_dev;
  const al_stub_model* m = static_cast<const al_stub_model*>(user);
  if (!m || !m->base_dev || !m->target_dev || m->vocab <= 0) return 1;
  if (n_rows <= 0) return 0;
  // the per-row local step sits right behind the row positions in the scheduler's upload buffer
  const int32_t* row_step_dev = row_pos_dev + n_rows;
  const long long total = (long long)n_rows * m->vocab;
  stub_model_kernel<<<(unsigned)((total + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
      m->base_dev, m->target_dev, m->gain, m->vocab, row_pos_dev, row_step_dev, n_rows, logits_dev);
  return cudaGetLastError() == cudaSuccess ? 0 : 2;
}

extern "C" al_status al_scheduler_run(al_handle* h, const al_sched_config* c, al_model_fn model, void* model_user,
                                      const al_sched_device_state* ds, const int32_t* prompt, int32_t* x_host,
                                      int32_t* output_host, int32_t* n_output, al_sched_lane* tree, int32_t max_tree,
                                      int32_t* n_tree, al_sched_stats* stats_out, void* stream) {
  const char* who = "al_scheduler_run";
  if (!h || !c || !model || !x_host || !output_host || !n_output || !tree || !n_tree || !stats_out)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL argument", who);
  if (c->prompt_len < 0 || c->gen_len <= 0 || c->block_size <= 0 || c->lookahead < 0 || c->lookahead > 0xffff ||
      c->vocab <= 0 || c->max_lane_steps <= 0 || c->max_iterations < 0 || c->refresh_period < 0 || c->refresh_margin < 0 ||
      c->n_delimiters < 0 || c->n_no_fork_prev < 0 || max_tree < 1 || c->mask_id < 0 || c->mask_id >= c->vocab ||
      c->eos_id >= c->vocab)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: bad configuration", who);
  if ((c->prompt_len > 0 && !prompt) || (c->n_delimiters > 0 && !c->delimiter_ids) ||
      (c->n_no_fork_prev > 0 && !c->no_fork_prev_ids))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL array with a positive count", who);
  al_status st = al_check_device(h, who);
  if (st != AL_OK) return st;
  const int P = c->prompt_len, L = c->gen_len, B = c->block_size, W = c->lookahead, V = c->vocab;
  const bool with_refresh = ds && ds->k_cache && ds->v_cache && ds->k_src && ds->v_src && c->refresh_period > 0;
  const bool with_attn = ds && ds->q && ds->k_new && ds->v_new && ds->out && ds->k_cache && ds->v_cache;
  if (ds && (with_refresh || with_attn)) {
    if ((st = al_check_shape(&ds->shape, who)) != AL_OK) return st;
    if (ds->shape.cache_rows < P + L) AL_FAIL(AL_ERR_INVALID_ARG, "%s: cache_rows %lld < P + L", who, (long long)ds->shape.cache_rows);
  }
  cudaStream_t cs = static_cast<cudaStream_t>(stream);

  // at most one generate lane is active at a time (a successor or continuation is created only when its parent stops
  // being active), refine lanes cover disjoint ranges: rows per iteration <= L + W
  const int rows_cap = L + W, lanes_cap = std::min(max_tree, L + 1);
  if (with_attn && ds->max_rows < rows_cap) AL_FAIL(AL_ERR_INVALID_ARG, "%s: device_state.max_rows %d < L + W = %d", who, ds->max_rows, rows_cap);
  Layout Y;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = al_round_up(off + bytes, 256); return o; };
  Y.lanes = take(sizeof(al_lane_desc) * lanes_cap);
  Y.tokens_in = take(4u * rows_cap);
  Y.row_pos = take(4u * 2 * rows_cap);                    // positions, then (right behind them) lane-local steps
  Y.row_step = Y.row_pos;                                 // (filled at row_pos + n_rows each iteration)
  Y.up_bytes = off;
  Y.down = off;
  Y.status = take(sizeof(al_lane_status_rec) * lanes_cap);
  Y.tokens_out = take(4u * rows_cap);
  Y.commit = take((size_t)rows_cap);
  Y.down_bytes = off - Y.down;
  Y.logits = take(sizeof(float) * (size_t)rows_cap * V);
  Y.conf = take(4u * rows_cap);
  Y.argmax = take(4u * rows_cap);
  Y.delims = take(4u * std::max(1, c->n_delimiters));
  Y.nofork = take(4u * std::max(1, c->n_no_fork_prev));
  Y.iota = take(4u * (size_t)(P + L));
  const size_t ws_attn_bytes = with_attn ? al_lane_attention_workspace_bytes(&ds->shape, lanes_cap, rows_cap, P + L) : 0;
  Y.ws_attn = take(ws_attn_bytes);
  Y.total = off;
  DeviceBuffers buf;
  AL_CUDA_OK(cudaMalloc(&buf.dev, Y.total));
  AL_CUDA_OK(cudaMallocHost(&buf.pinned, Y.logits));      // mirror of the upload + download regions
  uint8_t* D = buf.dev;
  uint8_t* Hp = buf.pinned;
  {                                                       // constants: id lists and the refresh position list 0..P+L-1
    std::vector<int32_t> iota((size_t)(P + L));
    for (int i = 0; i < P + L; ++i) iota[(size_t)i] = i;
    AL_CUDA_OK(cudaMemcpyAsync(D + Y.iota, iota.data(), 4u * iota.size(), cudaMemcpyHostToDevice, cs));
    if (c->n_delimiters) AL_CUDA_OK(cudaMemcpyAsync(D + Y.delims, c->delimiter_ids, 4u * c->n_delimiters, cudaMemcpyHostToDevice, cs));
    if (c->n_no_fork_prev) AL_CUDA_OK(cudaMemcpyAsync(D + Y.nofork, c->no_fork_prev_ids, 4u * c->n_no_fork_prev, cudaMemcpyHostToDevice, cs));
    AL_CUDA_OK(cudaStreamSynchronize(cs));                // the staging vector goes out of scope
  }

  for (int i = 0; i < P; ++i) x_host[i] = prompt[i];
  for (int i = 0; i < L; ++i) x_host[P + i] = c->mask_id;
  std::vector<al_sched_lane> nodes;
  std::vector<int> n_filled_of;                           // Eq.5 numerator of each node's last update
  auto new_node = [&](int role, int start, int len, int parent) {
    al_sched_lane n{};
    n.role = role; n.start = start; n.len = len; n.steps = 0; n.parent = parent;
    n.ref_child = n.gen_child = n.successor = -1; n.state = kActive; n.valid_prefix = 0; n.split_point = 0; n.n_masked = len;
    nodes.push_back(n); n_filled_of.push_back(0);
    return (int)nodes.size() - 1;
  };
  new_node(kGen, 0, std::min(B, L), -1);
  al_sched_stats S{};
  std::vector<int> active;

  while (S.iterations < c->max_iterations) {
    active.clear();
    for (int i = 0; i < (int)nodes.size(); ++i)
      if (nodes[(size_t)i].state == kActive) active.push_back(i);
    if (active.empty()) break;
    if ((int)active.size() > lanes_cap) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: %zu active lanes exceed the tree capacity %d", who, active.size(), max_tree);
    // ---- UPDATELANES (Alg.1 line 4): pack the active set, one model call, transfer, status ----
    al_lane_desc* lanes = reinterpret_cast<al_lane_desc*>(Hp + Y.lanes);
    int32_t* tok = reinterpret_cast<int32_t*>(Hp + Y.tokens_in);
    int32_t* pos = reinterpret_cast<int32_t*>(Hp + Y.row_pos);
    int n_rows = 0;
    for (size_t k = 0; k < active.size(); ++k) {
      const al_sched_lane& n = nodes[(size_t)active[k]];
      const int w = n.role == kGen ? std::min(W, L - (n.start + n.len)) : 0;
      n_rows += n.len + w;
    }
    if (n_rows > rows_cap) AL_FAIL(AL_ERR_UNSUPPORTED, "%s: %d rows in one iteration exceed L + W", who, n_rows);
    std::vector<int32_t> steps(active.size());
    int q_start = 0;
    for (size_t k = 0; k < active.size(); ++k) {
      const al_sched_lane& n = nodes[(size_t)active[k]];
      const int w = n.role == kGen ? std::min(W, L - (n.start + n.len)) : 0;
      lanes[k].group_id = 0; lanes[k].kv_base_row = 0; lanes[k].prefix_len = P + n.start;   // kappa_l: rows [0, P + s)
      lanes[k].q_start = q_start; lanes[k].q_len = n.len + w;
      lanes[k].flags = AL_LANE_FLAGS(n.role == kRef, w);
      steps[k] = n.steps;
      for (int i = 0; i < n.len + w; ++i) {
        tok[q_start + i] = x_host[P + n.start + i];
        pos[q_start + i] = n.start + i;
        pos[n_rows + q_start + i] = n.steps;              // lane-local step of the row, right behind the positions
      }
      q_start += n.len + w;
    }
    const int nl = (int)active.size();
    AL_CUDA_OK(cudaMemcpyAsync(D, Hp, Y.up_bytes, cudaMemcpyHostToDevice, cs));
    const al_lane_desc* lanes_dev = reinterpret_cast<const al_lane_desc*>(D + Y.lanes);
    const int32_t* tok_dev = reinterpret_cast<const int32_t*>(D + Y.tokens_in);
    float* logits_dev = reinterpret_cast<float*>(D + Y.logits);
    if (model(model_user, lanes, steps.data(), nl, n_rows, reinterpret_cast<const int32_t*>(D + Y.row_pos), tok_dev,
              logits_dev, stream) != 0)
      AL_FAIL(AL_ERR_CUDA, "%s: the model callback failed in iteration %d", who, S.iterations);
    if (with_attn) {                                      // the stub layer's attention over this iteration's lanes
      st = al_lane_attention(h, &ds->shape, ds->q, ds->k_new, ds->v_new, ds->k_cache, ds->v_cache, lanes_dev, nl, n_rows,
                             P + L, ds->out, nullptr, D + Y.ws_attn, ws_attn_bytes, stream);
      if (st != AL_OK) return st;
    }
    st = al_confidence_select(h, logits_dev, AL_F32, n_rows, V, V, tok_dev, c->mask_id, c->eos_id, c->tau, lanes_dev, nl,
                              AL_SELECT_FORCE_TOP1, reinterpret_cast<float*>(D + Y.conf),
                              reinterpret_cast<int32_t*>(D + Y.argmax), D + Y.commit,
                              reinterpret_cast<int32_t*>(D + Y.tokens_out), nullptr, 0, stream);
    if (st != AL_OK) return st;
    st = al_lane_status(h, lanes_dev, nl, n_rows, tok_dev, reinterpret_cast<const float*>(D + Y.conf),
                        reinterpret_cast<const int32_t*>(D + Y.argmax), c->mask_id, c->eos_id, c->tau_future,
                        reinterpret_cast<const int32_t*>(D + Y.delims), c->n_delimiters,
                        reinterpret_cast<const int32_t*>(D + Y.nofork), c->n_no_fork_prev, D + Y.commit,
                        reinterpret_cast<int32_t*>(D + Y.tokens_out), reinterpret_cast<al_lane_status_rec*>(D + Y.status),
                        stream);
    if (st != AL_OK) return st;
    AL_CUDA_OK(cudaMemcpyAsync(Hp + Y.down, D + Y.down, Y.down_bytes, cudaMemcpyDeviceToHost, cs));
    AL_CUDA_OK(cudaStreamSynchronize(cs));                // the one synchronisation of the iteration
    const al_lane_status_rec* status = reinterpret_cast<const al_lane_status_rec*>(Hp + Y.status);
    const int32_t* tok_out = reinterpret_cast<const int32_t*>(Hp + Y.tokens_out);
    for (size_t k = 0; k < active.size(); ++k) {          // write back (L80) and advance the lane clocks
      al_sched_lane& n = nodes[(size_t)active[k]];
      for (int i = 0; i < lanes[k].q_len; ++i) x_host[P + n.start + i] = tok_out[lanes[k].q_start + i];
      n.steps += 1;
      n.valid_prefix = status[k].valid_prefix; n.split_point = status[k].split_point; n.n_masked = status[k].n_masked;
      n_filled_of[(size_t)active[k]] = status[k].n_filled;
      S.tokens_committed += status[k].n_committed; S.tokens_drafted += status[k].n_drafts;
    }
    S.model_calls += 1; S.lane_forwards += nl; S.rows_forwarded += n_rows;
    // ---- Alg.1 lines 5-17: forks, completion, successors ----
    for (size_t k = 0; k < active.size(); ++k) {
      const int i = active[k];
      const bool done = nodes[(size_t)i].n_masked == 0 || nodes[(size_t)i].steps >= c->max_lane_steps;
      if (nodes[(size_t)i].role == kRef) {
        if (done) nodes[(size_t)i].state = kCompleted;
        continue;
      }
      const int s = nodes[(size_t)i].start, b = nodes[(size_t)i].len, p = nodes[(size_t)i].split_point,
                v = nodes[(size_t)i].valid_prefix;
      const bool fork = p > 0 && p < b && (double)n_filled_of[(size_t)i] >= (double)c->rho_min * b &&
                        nodes[(size_t)i].steps >= c->t_min && nodes[(size_t)i].n_masked > 0;
      if ((fork || (done && v > 0 && s + v < L)) && (int)nodes.size() + 2 > max_tree)
        AL_FAIL(AL_ERR_UNSUPPORTED, "%s: the lane tree outgrows max_tree = %d", who, max_tree);
      if (fork) {                                         // Eq.6: F(l, p) = (l_ref, l_gen)
        const int r = new_node(kRef, s, p, i);
        const int g = new_node(kGen, s + p, std::min(B, L - (s + p)), i);
        nodes[(size_t)i].ref_child = r; nodes[(size_t)i].gen_child = g; nodes[(size_t)i].state = kForked;
        S.forks += 1;
      } else if (done) {
        nodes[(size_t)i].state = kCompleted;
        if (v == 0 || s + v >= L) {                       // STOPADVANCE (Alg.1 line 13)
          S.stopped_frontiers += 1;
        } else {                                          // finalize the valid prefix, spawn the successor at s + v
          const int g = new_node(kGen, s + v, std::min(B, L - (s + v)), i);
          nodes[(size_t)i].successor = g;
          S.successors += 1;
        }
      }
    }
    S.iterations += 1;
    // ---- Eq.12: compact refresh of the meaningful prefix plus a margin ----
    if (c->refresh_period > 0 && S.iterations % c->refresh_period == 0) {
      int l_eff = 0;
      for (const al_sched_lane& n : nodes) l_eff = std::max(l_eff, n.start + n.valid_prefix);
      const int l_refresh = std::min(P + L, P + l_eff + c->refresh_margin);
      if (with_refresh) {
        st = al_kv_refresh(h, &ds->shape, ds->k_cache, ds->v_cache, ds->k_src, ds->v_src,
                           reinterpret_cast<const int32_t*>(D + Y.iota), l_refresh, 0, 1, 0, 0, stream);
        if (st != AL_OK) return st;
      }
      S.refreshes += 1; S.refreshed_rows_last = l_refresh;
    }
  }
  AL_CUDA_OK(cudaStreamSynchronize(cs));

  // ---- COLLECTDFS (L125): refine child before generate child; leaves cut at the first MASK (generate: or EOS) ----
  int n_out = 0;
  std::vector<int> stack{0};
  while (!stack.empty()) {
    const int i = stack.back();
    stack.pop_back();
    const al_sched_lane& n = nodes[(size_t)i];
    if (n.state == kForked) {
      stack.push_back(n.gen_child);                       // popped after the refine child
      stack.push_back(n.ref_child);
      continue;
    }
    for (int j = 0; j < n.len; ++j) {
      const int z = x_host[P + n.start + j];
      if (z == c->mask_id || (n.role == kGen && z == c->eos_id)) break;
      if (n_out < L) output_host[n_out++] = z;
    }
    if (n.successor >= 0) stack.push_back(n.successor);
  }
  *n_output = n_out;
  *n_tree = (int)nodes.size();
  for (size_t i = 0; i < nodes.size() && (int)i < max_tree; ++i) tree[i] = nodes[i];
  *stats_out = S;
  return AL_OK;
}
