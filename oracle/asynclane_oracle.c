/*
 * CPU ORACLE for the lane-batched denoising step of AsyncLane (arxiv 2606.08411).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.  It shares no code with the
 * CUDA path under paper_2606_08411_b200/csrc/ and is written as the plain definitions, in the
 * paper's order, with fp64 arithmetic on the (dtype-rounded) float32 inputs.
 *
 * The three functions of the lane step (O-A attention, O-B refresh, O-C confidence/select) are exact
 * definitions (lane batching "does not eliminate token-level computation, but replaces
 * serial lane forwards with grouped GPU execution"), so the oracle is the naive computation.  O-D (lane
 * status: Eq.4, 5, 8, 9) is integer bookkeeping written out from the equations.  Pins:
 * tests/test_oracle_pins*.py (brute force, closed forms, hand-worked examples under tests/golden/,
 * library special cases, invariants).  Nothing here is "parity unpinned".
 *
 * Lane descriptor (int32 x 6 per lane), after PAPER.md L56 Eq.1 / L70 / L168:
 *   [0] group_id     lanes of one shared-prefix group G_t (L168)
 *   [1] kv_base_row  first row of the lane's sequence in the cache pool
 *   [2] prefix_len   visible cache rows [kv_base_row, kv_base_row+prefix_len) = P + s_l (L70)
 *   [3] q_start      first row of the lane in the packed Q / K_new / V_new / logits
 *   [4] q_len        lane length b_l + w_l (L72 Eq.2)
 *   [5] flags        bit0 = refine lane (EOS suppressed, L80); bits 8..23 = lookahead window w_l (Eq.2):
 *                    the LAST w_l of the lane's q_len rows (only O-D distinguishes them)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * O-A  lane attention for ONE (lane, local row i, q-head h).
 * lane l is updated "using its own prefix state" kappa_l = cached KV "up to position
 * P + s_l"; L72-76 Eq.2-3: o_l = f_theta(u_l; kappa_l) over the lane's own tokens u_l; attention
 * is bidirectional (L24, L176).  So the key/value set of row i is
 *     cache rows kv_base_row + j, j in [0, prefix_len)   of kv-head g = h / n_rep
 *  ++ K_new/V_new rows q_start + j', j' in [0, q_len)    of kv-head g.
 * s_j = scale <q_i, k_j>;  p_j = exp(s_j - max)/Z;  O = sum_j p_j v_j;  LSE = max + ln Z.
 * Layouts: q [T][H_q][d]; k_new,v_new [T][H_kv][d]; caches [H_kv][cache_rows][d].
 * -----------------------------------------------------------------------------------------*/
void oracle_lane_attention_one(const float* q, const float* k_new, const float* v_new,
                               const float* k_cache, const float* v_cache, const int32_t* lane,
                               int local_row, int h, int n_q_heads, int n_kv_heads, int head_dim,
                               int64_t cache_rows, double scale, double* out_row, double* lse_out) {
  const int d = head_dim;
  const int n_rep = n_q_heads / n_kv_heads;
  const int g = h / n_rep;                       /* consecutive-repeat GQA mapping (reading C3) */
  const int64_t base = lane[1];
  const int prefix_len = lane[2], q_start = lane[3], q_len = lane[4];
  const int n_keys = prefix_len + q_len;
  const float* qi = q + ((int64_t)(q_start + local_row) * n_q_heads + h) * d;
  double* s = (double*)malloc(sizeof(double) * (size_t)(n_keys > 0 ? n_keys : 1));

  double m = -INFINITY;
  for (int j = 0; j < n_keys; ++j) {
    const float* kj = (j < prefix_len)
                          ? k_cache + ((int64_t)g * cache_rows + base + j) * d
                          : k_new + ((int64_t)(q_start + (j - prefix_len)) * n_kv_heads + g) * d;
    double acc = 0.0;
    for (int c = 0; c < d; ++c) acc += (double)qi[c] * (double)kj[c];
    s[j] = scale * acc;
    if (s[j] > m) m = s[j];
  }
  double Z = 0.0;
  for (int j = 0; j < n_keys; ++j) {
    s[j] = exp(s[j] - m);
    Z += s[j];
  }
  for (int c = 0; c < d; ++c) out_row[c] = 0.0;
  for (int j = 0; j < n_keys; ++j) {
    const float* vj = (j < prefix_len)
                          ? v_cache + ((int64_t)g * cache_rows + base + j) * d
                          : v_new + ((int64_t)(q_start + (j - prefix_len)) * n_kv_heads + g) * d;
    const double p = s[j] / Z;
    for (int c = 0; c < d; ++c) out_row[c] += p * (double)vj[c];
  }
  if (lse_out) *lse_out = m + log(Z);
  free(s);
}

/* All lanes, rows and heads: out [T][H_q][d] fp64, lse [T][H_q] fp64 (may be NULL). */
void oracle_lane_attention(const float* q, const float* k_new, const float* v_new,
                           const float* k_cache, const float* v_cache, const int32_t* lanes,
                           int n_lanes, int n_q_heads, int n_kv_heads, int head_dim,
                           int64_t cache_rows, double scale, double* out, double* lse) {
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int l = 0; l < n_lanes; ++l) {
    for (int h = 0; h < n_q_heads; ++h) {
      const int32_t* lane = lanes + 6 * l;
      for (int i = 0; i < lane[4]; ++i) {
        const int64_t row = (int64_t)(lane[3] + i) * n_q_heads + h;
        oracle_lane_attention_one(q, k_new, v_new, k_cache, v_cache, lane, i, h, n_q_heads,
                                  n_kv_heads, head_dim, cache_rows, scale, out + row * head_dim,
                                  lse ? lse + row : NULL);
      }
    }
  }
}

/* ------------------------------------------------------------------------------------------
 * O-B  compact cache refresh (Eq.12): the recomputed K/V rows of the
 * refreshed prefix positions overwrite the cache in place; every other byte is untouched.
 *   cache[layer][g][kv_base_row + pos[r]][:] = src[layer][r][g][:]      (K and V)
 * Pure byte copy: row_bytes = head_dim * element size.  Strides are in BYTES.
 * Precondition (reading C8): pos strictly increasing.
 * -----------------------------------------------------------------------------------------*/
void oracle_kv_refresh(uint8_t* k_cache, uint8_t* v_cache, const uint8_t* k_src,
                       const uint8_t* v_src, const int32_t* pos, int n_pos, int kv_base_row,
                       int n_layers, int n_kv_heads, int64_t cache_rows, int64_t row_bytes,
                       int64_t layer_stride_cache_bytes, int64_t layer_stride_src_bytes) {
  for (int layer = 0; layer < n_layers; ++layer)
    for (int r = 0; r < n_pos; ++r)
      for (int g = 0; g < n_kv_heads; ++g) {
        const int64_t dst = layer * layer_stride_cache_bytes +
                            ((int64_t)g * cache_rows + kv_base_row + pos[r]) * row_bytes;
        const int64_t src = layer * layer_stride_src_bytes + ((int64_t)r * n_kv_heads + g) * row_bytes;
        memcpy(k_cache + dst, k_src + src, (size_t)row_bytes);
        memcpy(v_cache + dst, v_src + src, (size_t)row_bytes);
      }
}

/* ------------------------------------------------------------------------------------------
 * O-C  confidence / argmax / threshold unmask select.
 * the first b_l logits update the lane "with the same confidence-based token
 * transfer rule as the underlying block-wise sampler"; L108 Eq.8 names the quantities: greedy
 * token x^_i = argmax_v o_iv and confidence q_i = softmax probability of x^_i, compared with >=.
 * L80: refine lanes suppress EOS; committed tokens are written back.
 * Readings: C4 commit iff masked AND q_i >= tau;  C5 refine-lane rows set
 * logit[eos] = -inf before softmax and argmax;  C6 the FIRST index attaining the max wins;
 * force-top1 (flags bit0): a lane with masked rows but no commit commits its masked row of
 * largest confidence (lowest row on ties).
 * Outputs per row: conf, argmax, p2 (second-largest probability, for the tie exemption of the
 * parity tests), commit, tokens_out.  lanes may be NULL (one implicit generate lane over all rows).
 * -----------------------------------------------------------------------------------------*/
void oracle_confidence_select(const float* logits, int n_rows, int vocab, int64_t row_stride,
                              const int32_t* tokens_in, int mask_id, int eos_id, double threshold,
                              const int32_t* lanes, int n_lanes, int flags, double* conf,
                              int32_t* argmax, double* p2, uint8_t* commit, int32_t* tokens_out) {
  /* row -> suppress-EOS flag from the lane descriptors */
  uint8_t* suppress = (uint8_t*)calloc((size_t)(n_rows > 0 ? n_rows : 1), 1);
  if (lanes && eos_id >= 0)
    for (int l = 0; l < n_lanes; ++l)
      if (lanes[6 * l + 5] & 1)
        for (int i = 0; i < lanes[6 * l + 4]; ++i) {
          const int row = lanes[6 * l + 3] + i;
          if (row >= 0 && row < n_rows) suppress[row] = 1;
        }

#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < n_rows; ++i) {
    const float* x = logits + (int64_t)i * row_stride;
    const int sup = suppress[i] ? eos_id : -1;
    int a = -1;
    double m = -INFINITY;
    for (int v = 0; v < vocab; ++v) {
      const double xv = (v == sup) ? -INFINITY : (double)x[v];
      if (a < 0 || xv > m) { m = xv; a = v; }          /* strict > keeps the first maximiser */
    }
    double Z = 0.0, second = -INFINITY;
    for (int v = 0; v < vocab; ++v) {
      const double xv = (v == sup) ? -INFINITY : (double)x[v];
      Z += exp(xv - m);
      if (v != a && xv > second) second = xv;
    }
    conf[i] = 1.0 / Z;
    argmax[i] = a;
    if (p2) p2[i] = (vocab > 1) ? exp(second - m) / Z : 0.0;
    commit[i] = (uint8_t)(tokens_in[i] == mask_id && conf[i] >= threshold);
  }

  if (flags & 1) {                                        /* force-top1 per lane */
    const int32_t whole[6] = {0, 0, 0, 0, n_rows, 0};
    const int nl = lanes ? n_lanes : 1;
    for (int l = 0; l < nl; ++l) {
      const int32_t* lane = lanes ? lanes + 6 * l : whole;
      int any_masked = 0, any_commit = 0, best = -1;
      for (int i = 0; i < lane[4]; ++i) {
        const int row = lane[3] + i;
        if (row < 0 || row >= n_rows) continue;
        if (tokens_in[row] == mask_id) {
          any_masked = 1;
          if (best < 0 || conf[row] > conf[best]) best = row;
        }
        if (commit[row]) any_commit = 1;
      }
      if (any_masked && !any_commit) commit[best] = 1;
    }
  }
  for (int i = 0; i < n_rows; ++i) tokens_out[i] = commit[i] ? argmax[i] : tokens_in[i];
  free(suppress);
}

/* ------------------------------------------------------------------------------------------
 * O-D  lane status after the transfer: the per-lane integers the host
 * scheduler (Alg.1) needs from one iteration, and the lookahead draft rule.
 *
 * A lane's rows are u_l = [z_l ; lookahead window] (Eq.2): the first b = q_len - w rows are
 * the lane state z_l, the last w rows the lookahead window; w = (flags >> 8) & 0xffff.
 *
 *  Eq.8 (L108)  lookahead rows:  x_i <- x^_i  if  x_i = [MASK], q_i >= tau_future, x^_i not in E
 *               (E = {EOS}; the rows are decided here whatever the transfer rule wrote for them)
 *  Eq.5 (L91)   n_filled    = |{ i < b : z_i != [MASK] }|           (fill ratio = n_filled / b)
 *  Eq.9 (L113)  valid_prefix v_l = min( { i : z_i = [MASK] or z_i in E } U { b } ),  i 0-based
 *               (the paper's i - 1 with 1-based i)
 *  Eq.4 (L86)   split_point p_l = 1 + max{ i : z_i in D_task and ValidBoundary(z_{1:i}) }, i.e.
 *               with 0-based i the number of tokens up to and including the last valid delimiter;
 *               0 when there is none.  ValidBoundary (reading C17): a delimiter whose PREVIOUS token is
 *               in the no-fork set does not count (L195 "numeric-period patterns excluded": a period
 *               after a digit token); the first token of a lane has no previous token.
 *  n_committed = rows of z_l committed in this iteration, n_drafts = lookahead rows drafted,
 *  n_masked = b - n_filled.
 * All of z is read AFTER the transfer (tokens_io holds tokens_out of the select on entry).
 * status: int32 [n_lanes][8] = {n_filled, valid_prefix, split_point, n_committed, n_drafts, n_masked, 0, 0}.
 * -----------------------------------------------------------------------------------------*/
void oracle_lane_status(const int32_t* lanes, int n_lanes, int n_rows, const int32_t* tokens_in,
                        const double* conf, const int32_t* argmax, int mask_id, int eos_id,
                        double tau_future, const int32_t* delimiters, int n_delimiters,
                        const int32_t* no_fork_prev, int n_no_fork_prev, uint8_t* commit_io,
                        int32_t* tokens_io, int32_t* status) {
  for (int l = 0; l < n_lanes; ++l) {
    const int32_t* lane = lanes + 6 * l;
    const int q_start = lane[3], q_len = lane[4];
    int w = (lane[5] >> 8) & 0xffff;
    if (w > q_len) w = q_len;
    const int b = q_len - w;
    int32_t* st = status + 8 * l;
    for (int k = 0; k < 8; ++k) st[k] = 0;
    /* Eq.8: the lookahead window */
    for (int i = b; i < q_len; ++i) {
      const int row = q_start + i;
      if (row < 0 || row >= n_rows) continue;
      const int c = tokens_in[row] == mask_id && conf[row] >= tau_future && argmax[row] != eos_id;
      commit_io[row] = (uint8_t)c;
      tokens_io[row] = c ? argmax[row] : tokens_in[row];
      st[4] += c;
    }
    /* the lane state z_l after the transfer */
    int v = b, p = 0;
    for (int i = 0; i < b; ++i) {
      const int row = q_start + i;
      const int z = tokens_io[row];
      if (z != mask_id) st[0] += 1;
      if (commit_io[row]) st[3] += 1;
      if ((z == mask_id || z == eos_id) && i < v) v = i;
      int is_delim = 0;
      for (int d = 0; d < n_delimiters; ++d) is_delim |= (z == delimiters[d]);
      if (is_delim) {
        int ok = 1;
        if (i > 0)
          for (int d = 0; d < n_no_fork_prev; ++d) ok &= (tokens_io[row - 1] != no_fork_prev[d]);
        if (ok) p = i + 1;
      }
    }
    st[1] = v;
    st[2] = p;
    st[5] = b - st[0];
  }
}

/* ------------------------------------------------------------------------------------------
 * O-E  refresh forward (Eq.12): the prefix states of a range are
 * RECOMPUTED -- bidirectional attention of the range's rows over [older prefix ; the range itself]
 * (Eq.2-3 with the range as the "lane") -- and the recomputed K/V rows are written into the cache right
 * behind that older prefix:
 *     out, lse        = O-A on the same arguments (the cache is read BEFORE it is written)
 *     cache[g][kv_base_row + prefix_len + i][:] = k_new[q_start + i][g][:]   for i in [0, q_len)   (K and V)
 * Eq.12's own case is prefix_len = 0, q_len = L_refresh: dense self-attention over the refreshed range whose
 * states replace cache rows [0, L_refresh).  The same call with prefix_len > 0 is the "finalize the valid
 * prefix" append of Alg.1 line 16.  Caches are float32 here (values already rounded to the I/O dtype).
 * -----------------------------------------------------------------------------------------*/
void oracle_refresh_forward(const float* q, const float* k_new, const float* v_new, float* k_cache, float* v_cache,
                            const int32_t* lanes, int n_lanes, int n_q_heads, int n_kv_heads, int head_dim,
                            int64_t cache_rows, double scale, double* out, double* lse) {
  oracle_lane_attention(q, k_new, v_new, k_cache, v_cache, lanes, n_lanes, n_q_heads, n_kv_heads, head_dim, cache_rows,
                        scale, out, lse);
  for (int l = 0; l < n_lanes; ++l) {
    const int32_t* lane = lanes + 6 * l;
    for (int i = 0; i < lane[4]; ++i)
      for (int g = 0; g < n_kv_heads; ++g) {
        const int64_t dst = ((int64_t)g * cache_rows + lane[1] + lane[2] + i) * head_dim;
        const int64_t src = ((int64_t)(lane[3] + i) * n_kv_heads + g) * head_dim;
        memcpy(k_cache + dst, k_new + src, sizeof(float) * (size_t)head_dim);
        memcpy(v_cache + dst, v_new + src, sizeof(float) * (size_t)head_dim);
      }
  }
}

/* ------------------------------------------------------------------------------------------
 * O-F  LM head fused with the transfer rule (the step upstream of PAPER.md L78:
 * "the first b_l logits of o_l are used to update the current lane"): the logits of row i are
 *     o_iv = sum_k hidden[i][k] * weight[v][k]            (weight stored [V][K] as a linear layer keeps it)
 * and are consumed by exactly the rule of O-C (first argmax, q = 1 / sum_v exp(o_v - max), EOS = -inf on
 * refine-lane rows, commit iff MASK and q >= tau, optional force-top1) WITHOUT ever being stored as an
 * [N][V] array by the product.  Here they are formed in fp64, one row at a time, and fed through the same
 * steps in the same order as O-C.
 * -----------------------------------------------------------------------------------------*/
void oracle_lm_head_confidence(const float* hidden, const float* weight, int n_rows, int vocab, int hidden_dim,
                               const int32_t* tokens_in, int mask_id, int eos_id, double threshold,
                               const int32_t* lanes, int n_lanes, int flags, double* conf, int32_t* argmax,
                               double* p2, uint8_t* commit, int32_t* tokens_out) {
  uint8_t* suppress = (uint8_t*)calloc((size_t)(n_rows > 0 ? n_rows : 1), 1);
  if (lanes && eos_id >= 0)
    for (int l = 0; l < n_lanes; ++l)
      if (lanes[6 * l + 5] & 1)
        for (int i = 0; i < lanes[6 * l + 4]; ++i) {
          const int row = lanes[6 * l + 3] + i;
          if (row >= 0 && row < n_rows) suppress[row] = 1;
        }
#pragma omp parallel
  {
    double* x = (double*)malloc(sizeof(double) * (size_t)vocab);
#pragma omp for schedule(dynamic, 1)
    for (int i = 0; i < n_rows; ++i) {
      const float* h = hidden + (int64_t)i * hidden_dim;
      for (int v = 0; v < vocab; ++v) {
        const float* w = weight + (int64_t)v * hidden_dim;
        double acc = 0.0;
        for (int k = 0; k < hidden_dim; ++k) acc += (double)h[k] * (double)w[k];
        x[v] = acc;
      }
      if (suppress[i]) x[eos_id] = -INFINITY;
      int a = -1;
      double m = -INFINITY;
      for (int v = 0; v < vocab; ++v)
        if (a < 0 || x[v] > m) { m = x[v]; a = v; }        /* strict > keeps the first maximiser */
      double Z = 0.0, second = -INFINITY;
      for (int v = 0; v < vocab; ++v) {
        Z += exp(x[v] - m);
        if (v != a && x[v] > second) second = x[v];
      }
      conf[i] = 1.0 / Z;
      argmax[i] = a;
      if (p2) p2[i] = (vocab > 1) ? exp(second - m) / Z : 0.0;
      commit[i] = (uint8_t)(tokens_in[i] == mask_id && conf[i] >= threshold);
    }
    free(x);
  }
  if (flags & 1) {                                        /* force-top1 per lane, as in O-C */
    const int32_t whole[6] = {0, 0, 0, 0, n_rows, 0};
    const int nl = lanes ? n_lanes : 1;
    for (int l = 0; l < nl; ++l) {
      const int32_t* lane = lanes ? lanes + 6 * l : whole;
      int any_masked = 0, any_commit = 0, best = -1;
      for (int i = 0; i < lane[4]; ++i) {
        const int row = lane[3] + i;
        if (row < 0 || row >= n_rows) continue;
        if (tokens_in[row] == mask_id) {
          any_masked = 1;
          if (best < 0 || conf[row] > conf[best]) best = row;
        }
        if (commit[row]) any_commit = 1;
      }
      if (any_masked && !any_commit) commit[best] = 1;
    }
  }
  for (int i = 0; i < n_rows; ++i) tokens_out[i] = commit[i] ? argmax[i] : tokens_in[i];
  free(suppress);
}
