/*
 * asynclane.h -- C ABI of the B200 (sm_100a) lane-batched denoising step of AsyncLane
 * (arxiv 2606.08411).  Citations "P:L<n>" are lines of the paper text.
 *
 * One scheduler iteration (Alg.1 UPDATELANES) runs, per shared-prefix group, one batched
 * model call (Eq.11).  This library is the data-parallel part of that call:
 *
 *   al_lane_attention     shared-prefix lane-batched bidirectional attention   (Eq.2-3)
 *   al_kv_refresh         compact cache refresh: in-place K/V row scatter       (Eq.12)
 *   al_confidence_select  softmax confidence / argmax / threshold unmask select (Eq.8)
 *
 * Conventions
 *  - Every pointer named *_dev (and q/k/v/caches/logits/outputs/workspace) is a DEVICE pointer owned
 *    by the caller; the library never allocates or frees device memory on the hot path and keeps no
 *    reference after the call returns.  `al_handle` owns only small host-side state (device id, SM
 *    count, tensor-map encoder entry point).
 *  - Every hot call only ENQUEUES work on `cuda_stream` (a cudaStream_t passed as void*): no device
 *    synchronisation, no host read of device descriptors; all calls are CUDA-graph capturable.
 *  - Every call returns an al_status; nothing throws.  On error nothing has been launched, except
 *    AL_ERR_CUDA which reports a failed launch or copy.  The calling thread's current CUDA device
 *    must be the handle's device (al_create does not change it); otherwise AL_ERR_INVALID_ARG.  `al_last_error()` gives a thread-local message.
 *  - Sizes of 0 lanes / 0 positions / 0 rows are valid no-ops returning AL_OK.
 *  - 16-byte alignment is required of q, k_new, v_new, caches, out, k_src, v_src, logits rows
 *    (row_stride * element size % 16 == 0 for the vector path; otherwise a scalar path is used)
 *    and of the workspace.
 */
#ifndef ASYNCLANE_H_
#define ASYNCLANE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  AL_OK = 0,
  AL_ERR_INVALID_ARG = 1, /* null pointer, negative size, misaligned pointer, bad enum            */
  AL_ERR_UNSUPPORTED = 2, /* valid request this build has no kernel for (e.g. head_dim, dtype)    */
  AL_ERR_WORKSPACE = 3,   /* workspace_bytes smaller than al_*_workspace_bytes() for these bounds */
  AL_ERR_CUDA = 4         /* a CUDA runtime / driver call failed; see al_last_error()             */
} al_status;

typedef enum { AL_F32 = 0, AL_BF16 = 1 } al_dtype;

typedef struct al_handle al_handle; /* opaque */

/*
 * Lane descriptor: one per active lane l = (r_l, s_l, b_l, z_l, t_l) of Eq.1, reduced to
 * what the kernels need.  The array lives in DEVICE memory so that a captured graph can be
 * replayed with new lanes.  Six int32, 24 bytes, no padding.
 */
typedef struct {
  int32_t group_id;    /* lanes of one shared-prefix group G_t share one prefix KV         */
  int32_t kv_base_row; /* "prefix offset": first row of this lane's sequence in the cache pool      */
  int32_t prefix_len;  /* visible cache rows [kv_base_row, kv_base_row+prefix_len) = P+s_l  */
  int32_t q_start;     /* "lane start": first row of the lane in packed Q/K_new/V_new/O/logits      */
  int32_t q_len;       /* "lane length": b_l + w_l rows of u_l (Eq.2)                         */
  int32_t flags;       /* bit0: refine lane => EOS suppressed in confidence_select;
                          bits 8..23: lookahead window w_l (Eq.2), the LAST w_l of the q_len rows */
} al_lane_desc;

#define AL_LANE_FLAG_REFINE 1
#define AL_LANE_LOOKAHEAD(flags) (((flags) >> 8) & 0xffff)
#define AL_LANE_FLAGS(refine, lookahead) (((refine) ? AL_LANE_FLAG_REFINE : 0) | (((lookahead) & 0xffff) << 8))

typedef struct {
  int32_t n_q_heads;  /* H_q                                                            */
  int32_t n_kv_heads; /* H_kv, divides H_q; q-head h reads kv-head h / (H_q/H_kv)        */
  int32_t head_dim;   /* d: bf16 tensor-core path needs 128 (64 also built); f32: <= 256 */
  int32_t dtype;      /* al_dtype of q, k_new, v_new, caches and out                     */
  int64_t cache_rows; /* capacity in rows of ONE kv-head plane of the cache pool         */
  float scale;        /* softmax scale; 0 => 1/sqrt(head_dim) (paper silent)             */
  int32_t reserved;   /* must be 0                                                       */
} al_attn_shape;

/* ---- life cycle ------------------------------------------------------------------------------- */

/* Creates a handle bound to CUDA device `device` (queries SM count, resolves the tensor-map encoder).
 * Fails with AL_ERR_CUDA when no usable device exists: there is no CPU fallback.
 * Two environment switches are read here, once, for tests and measurements (results are the same either way):
 * ASYNCLANE_SELF_PLAN=0 (small attention calls launch the plan kernel too) and ASYNCLANE_CONF_SPREAD=0
 * (confidence launches of less than one resident wave do not cap the CTAs per SM). */
al_status al_create(al_handle** out_handle, int device);
al_status al_destroy(al_handle* handle);
/* Thread-local, never NULL, valid until the next failing call on this thread. */
const char* al_last_error(void);
/* "asynclane-b200 <version> sm_100a" */
const char* al_version(void);
/* Number of SMs of the handle's device (grid sizing information for callers / bench). */
int32_t al_sm_count(const al_handle* handle);

/* ---- (a) shared-prefix lane-batched attention ------------------------------------------------- */

/*
 * For every lane l, q-head h (kv-head g = h / n_rep) and local row i in [0, q_len):
 *   keys/values = cache rows kv_base_row + j, j in [0, prefix_len)      (plane g of k_cache/v_cache)
 *              ++ k_new/v_new rows q_start + j', j' in [0, q_len)        (the lane's own rows)
 *   out[q_start+i][h][:] = softmax_j(scale * <q_i, k_j>) . v_j           (bidirectional, no causal mask)
 *   lse[q_start+i][h]    = log sum_j exp(scale * <q_i, k_j>)             (optional)
 * Lanes never see each other ("updated independently using its own prefix state"); lanes with
 * equal group_id address the same cache rows, which the kernel reads from HBM once per group and
 * kv-head, not once per lane.
 *
 * Layouts (row-major, innermost last):
 *   q, out        [T][H_q][d]        T = total packed rows (sum of q_len)
 *   k_new, v_new  [T][H_kv][d]
 *   k_cache, v_cache [H_kv][cache_rows][d]     (never written by this call)
 *   lse_or_null   float [T][H_q]
 * Host-side bounds: n_lanes (exact), total_q_rows = T (exact), max_prefix_len >= every prefix_len.
 * Preconditions on lanes_dev (not checked on the hot path; see al_validate_lanes): lanes are disjoint
 * in [q_start, q_start+q_len), 0 <= kv_base_row, kv_base_row+prefix_len <= cache_rows, q_len >= 1.
 * Lanes of one group that are adjacent in the array and contiguous in q_start are stacked into
 * common 128-row tensor-core tiles.
 * Limits of the tensor-core path (bf16, head_dim 128): at most 1024 lanes per call and at most 2048
 * query tiles (ceil(total_q_rows / (2 * floor(128 / n_rep))) + n_lanes); beyond them AL_ERR_UNSUPPORTED.
 * Results are deterministic: the same inputs give bit-identical outputs from call to call.
 * Rows of Q not covered by any lane are not written in `out`.
 * Finite-input contract (reading C14): every row of q, k_new and v_new in [0, total_q_rows) and every
 * cache row that SOME lane of the call may see must hold finite values -- lanes share 128-row tensor-core
 * tiles, so a NaN/Inf in one lane's K_new/V_new rows reaches the rows stacked with it (0 x NaN).  Cache rows
 * that NO lane sees (beyond the longest prefix_len of the lanes addressing that region: unwritten or
 * recycled memory) may hold anything, NaN included: their scores are masked by selection and the V
 * rows the last key tile rounds up to are zeroed on chip before the tensor core reads them.
 */
size_t al_lane_attention_workspace_bytes(const al_attn_shape* shape, int32_t n_lanes,
                                         int32_t total_q_rows, int32_t max_prefix_len);
al_status al_lane_attention(al_handle* handle, const al_attn_shape* shape, const void* q,
                            const void* k_new, const void* v_new, const void* k_cache,
                            const void* v_cache, const al_lane_desc* lanes_dev, int32_t n_lanes,
                            int32_t total_q_rows, int32_t max_prefix_len, void* out,
                            float* lse_or_null, void* workspace, size_t workspace_bytes,
                            void* cuda_stream);

/*
 * The work decomposition of al_lane_attention (tiles, key ranges, per-CTA work lists) depends only
 * on the lane descriptors, not on the layer: one scheduler iteration (P:L135 UPDATELANES) calls the
 * model once per group (Eq.11) and every layer of that call sees the same lanes.
 *   al_lane_plan               builds the decomposition from lanes_dev into `workspace` (one small launch)
 *   al_lane_attention_planned  runs the attention of one layer from a workspace al_lane_plan filled
 *                              with the SAME shape, lanes_dev contents, n_lanes, total_q_rows and
 *                              max_prefix_len
 * Small calls need no plan launch at all: with at most 32 lanes, (ceil(total_q_rows / floor(128 / n_rep)) +
 * n_lanes - 1) * H_kv <= SMs and ceil(max_prefix_len / 64) + ceil(total_q_rows / 64) <= 24, every CTA of the
 * attention kernel derives its own work from lanes_dev in its prologue (the same decomposition the plan
 * launch would write); al_lane_plan then enqueues nothing and leaves the workspace untouched.  The rule
 * depends on the host-side bounds only, which is why the planned call must be given the same ones.  (A
 * handle created while the environment holds ASYNCLANE_SELF_PLAN=0 always launches the plan.)
 * al_lane_attention == al_lane_plan followed by al_lane_attention_planned.  The planned call leaves
 * the plan intact, so it may be repeated (other layers, other q/k/v/cache/out pointers) on the same
 * stream.  For shapes the tensor-core path does not cover (fp32, head_dim != 128) there is no plan:
 * al_lane_plan is a no-op and al_lane_attention_planned runs the plain-ALU kernel.
 */
al_status al_lane_plan(al_handle* handle, const al_attn_shape* shape, const al_lane_desc* lanes_dev,
                       int32_t n_lanes, int32_t total_q_rows, int32_t max_prefix_len, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);
al_status al_lane_attention_planned(al_handle* handle, const al_attn_shape* shape, const void* q,
                                    const void* k_new, const void* v_new, const void* k_cache,
                                    const void* v_cache, const al_lane_desc* lanes_dev,
                                    int32_t n_lanes, int32_t total_q_rows, int32_t max_prefix_len,
                                    void* out, float* lse_or_null, void* workspace,
                                    size_t workspace_bytes, void* cuda_stream);

/* ---- (b) compact cache refresh ---------------------------------------------------------------- */

/*
 * For r in [0, n_pos), layer in [0, n_layers), kv-head g:
 *   k_cache[layer][g][kv_base_row + pos[r]][:] = k_src[layer][r][g][:]     (same for V)
 * Bit copy; every other byte of the caches is untouched.  Layouts: caches [H_kv][cache_rows][d] per
 * layer, layers `layer_stride_cache` ELEMENTS apart; src [R][H_kv][d] per layer, layers
 * `layer_stride_src` elements apart.  Precondition: pos strictly increasing (unique), each
 * kv_base_row + pos[r] in [0, cache_rows).  Duplicates make the result order-dependent; the hot call
 * cannot check device-resident positions without synchronising -- al_validate_refresh does.
 * head_dim * element size must be a multiple of 16.
 */
al_status al_kv_refresh(al_handle* handle, const al_attn_shape* shape, void* k_cache, void* v_cache,
                        const void* k_src, const void* v_src, const int32_t* pos_dev, int32_t n_pos,
                        int32_t kv_base_row, int32_t n_layers, int64_t layer_stride_cache,
                        int64_t layer_stride_src, void* cuda_stream);

/*
 * Refresh forward (Eq.12): the prefix states of a range are recomputed and
 * replace the cached ones.  Each descriptor is one RANGE: its q_len rows (q, k_new, v_new: the recomputed
 * activations of this layer) attend bidirectionally to [the older prefix the range keeps: cache rows
 * kv_base_row + [0, prefix_len) ; the range itself] exactly as in al_lane_attention, and then
 *   k_cache[g][kv_base_row + prefix_len + i][:] = k_new[q_start + i][g][:]      (same for V), i in [0, q_len)
 * Eq.12's own case is prefix_len = 0, q_len = L_refresh (dense self-attention over the refreshed range); with
 * prefix_len > 0 the same call appends a finalized valid prefix (Alg.1 line 16).  The attention reads the
 * cache BEFORE these rows are written (stream order); kv_base_row + prefix_len + q_len <= cache_rows, and
 * the ranges of one call must write disjoint cache rows (two ranges appending to the same rows race).
 * Arguments, limits and workspace as al_lane_attention (max_prefix_len >= every prefix_len).
 */
al_status al_refresh_forward(al_handle* handle, const al_attn_shape* shape, const void* q,
                             const void* k_new, const void* v_new, void* k_cache, void* v_cache,
                             const al_lane_desc* lanes_dev, int32_t n_lanes, int32_t total_q_rows,
                             int32_t max_prefix_len, void* out, float* lse_or_null, void* workspace,
                             size_t workspace_bytes, void* cuda_stream);

/* ---- (c) confidence / argmax / threshold select ----------------------------------------------- */

#define AL_SELECT_FORCE_TOP1 1

/*
 * Per row i of logits [n_rows][vocab] (row_stride elements between rows):
 *   x = logits row (refine-lane rows with eos_id >= 0: x[eos_id] = -inf)
 *   argmax_out[i] = first index attaining max x;  conf_out[i] = 1 / sum_v exp(x_v - max x)
 *   commit_out[i] = (tokens_in[i] == mask_id) && conf_out[i] >= threshold
 *   flags & AL_SELECT_FORCE_TOP1: a lane with masked rows but no commit commits its masked row of
 *     largest confidence (lowest row on ties).  Without lanes, all rows form one generate lane.
 *   tokens_out[i] = commit ? argmax : tokens_in[i]     (tokens_out may alias tokens_in)
 * conf is computed in fp32 from the dtype-rounded logits.  Rows must hold at least one finite value.
 * No workspace is needed (partials are merged on chip through cluster shared memory):
 * al_confidence_select_workspace_bytes returns 0 and `workspace` may be NULL; both stay in the
 * signature so that callers size arenas through one query per call.
 */
size_t al_confidence_select_workspace_bytes(int32_t n_rows, int32_t vocab);
al_status al_confidence_select(al_handle* handle, const void* logits, int32_t logits_dtype,
                               int32_t n_rows, int32_t vocab, int64_t row_stride,
                               const int32_t* tokens_in_dev, int32_t mask_id, int32_t eos_id,
                               float threshold, const al_lane_desc* lanes_dev_or_null,
                               int32_t n_lanes, int32_t flags, float* conf_out, int32_t* argmax_out,
                               uint8_t* commit_out, int32_t* tokens_out, void* workspace,
                               size_t workspace_bytes, void* cuda_stream);

/*
 * LM head fused with the transfer rule (the step upstream of P:L78): the logits
 *   o[i][v] = sum_k hidden[i][k] * weight[v][k]          hidden [n_rows][hidden_dim], weight [vocab][hidden_dim],
 * both bf16 row-major (the layout a linear layer keeps), fp32 accumulation on the tensor cores, are consumed
 * tile by tile by the recurrence of al_confidence_select and never stored: outputs, EOS suppression on refine
 * lanes, commit rule and AL_SELECT_FORCE_TOP1 are exactly those of al_confidence_select (argmax = first
 * maximiser of the fp32 logits).  hidden_dim must be a multiple of 8; any n_rows, vocab.  The workspace
 * (al_lm_head_confidence_workspace_bytes) holds one (m, s, idx) per row and vocabulary chunk; no zeroing needed.
 * With few rows (<= 512) the call streams the weights once at HBM rate; with many it is bound by the tensor
 * cores' operand traffic through L2 (single-CTA 128 x 256 tiles) -- see DESIGN.md K5.
 */
size_t al_lm_head_confidence_workspace_bytes(int32_t n_rows, int32_t vocab);
al_status al_lm_head_confidence(al_handle* handle, const void* hidden_bf16, const void* weight_bf16,
                                int32_t n_rows, int32_t vocab, int32_t hidden_dim,
                                const int32_t* tokens_in_dev, int32_t mask_id, int32_t eos_id, float threshold,
                                const al_lane_desc* lanes_dev_or_null, int32_t n_lanes, int32_t flags,
                                float* conf_out, int32_t* argmax_out, uint8_t* commit_out, int32_t* tokens_out,
                                void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The same call for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): it takes no workspace -- the partials live in a device array of
 * AL_LM_HEAD_STATIC_SCRATCH_BYTES (1 MiB) that is part of the library image, so every GPU that loads the library
 * holds it until exit -- and calls no cudaMalloc / cudaFree or allocating library routine.  Arguments, results and
 * errors as al_lm_head_confidence; additionally AL_ERR_UNSUPPORTED, before anything is enqueued, when the shape
 * needs more scratch than the array holds (16 bytes x 128 x ceil(n_rows / 128) x vocabulary chunks, the chunks
 * chosen from the SM count: 128 x 126464 takes 0.3 MB, 3264 x 152064 0.9 MB, 8192 x 152064 2 MB -- too many).
 * ALL calls on a device share the one array: calls that may overlap on the GPU (different streams, or graphs
 * replayed concurrently) race on it and must be serialised by the caller; calls on one stream are ordered.
 * The array keeps the last call's contents; nothing in it has to be cleared (every slot read is written first).
 */
#define AL_LM_HEAD_STATIC_SCRATCH_BYTES (1 << 20)
size_t al_lm_head_confidence_static_max_bytes(void);
al_status al_lm_head_confidence_static(al_handle* handle, const void* hidden_bf16, const void* weight_bf16,
                                       int32_t n_rows, int32_t vocab, int32_t hidden_dim,
                                       const int32_t* tokens_in_dev, int32_t mask_id, int32_t eos_id, float threshold,
                                       const al_lane_desc* lanes_dev_or_null, int32_t n_lanes, int32_t flags,
                                       float* conf_out, int32_t* argmax_out, uint8_t* commit_out, int32_t* tokens_out,
                                       void* cuda_stream);

/* ---- (d) lane status: what the scheduler reads back from one iteration ------------------------- */

/*
 * Per lane, AFTER the transfer.  A lane's rows are u_l = [z_l ; lookahead window]
 * (Eq.2): the first b = q_len - w rows are the lane state z_l, the last w = AL_LANE_LOOKAHEAD(flags)
 * rows the window.
 *   lookahead rows (Eq.8): commit_io[i] = tokens_in[i] == mask_id && conf[i] >= tau_future &&
 *     argmax[i] != eos_id;  tokens_io[i] = commit ? argmax[i] : tokens_in[i]   (this call DECIDES those rows,
 *     whatever al_confidence_select wrote for them)
 *   n_filled     |{ i < b : z_i != MASK }|                       (Eq.5: fill ratio = n_filled / b)
 *   valid_prefix v_l = first 0-based i with z_i == MASK or z_i == eos_id, else b          (Eq.9)
 *   split_point  p_l = 1 + the last 0-based i < b with z_i in delimiter_ids and ValidBoundary, else 0
 *                (Eq.4).  ValidBoundary (reading C17): the delimiter's previous token (i > 0) is not
 *                in no_fork_prev_ids -- the "numeric-period patterns excluded" of P:L195
 *   n_committed  rows of z_l with commit_io set;  n_drafts  lookahead rows drafted;  n_masked = b - n_filled
 * z is read from tokens_io (on entry the tokens_out of al_confidence_select; must not alias tokens_in).
 * One small launch, no synchronisation; status_out_dev[n_lanes] is what the host copies back.
 */
typedef struct {
  int32_t n_filled, valid_prefix, split_point, n_committed, n_drafts, n_masked, reserved[2];
} al_lane_status_rec;

al_status al_lane_status(al_handle* handle, const al_lane_desc* lanes_dev, int32_t n_lanes, int32_t n_rows,
                         const int32_t* tokens_in_dev, const float* conf_dev, const int32_t* argmax_dev,
                         int32_t mask_id, int32_t eos_id, float tau_future,
                         const int32_t* delimiter_ids_dev, int32_t n_delimiters,
                         const int32_t* no_fork_prev_ids_dev, int32_t n_no_fork_prev,
                         uint8_t* commit_io_dev, int32_t* tokens_io_dev,
                         al_lane_status_rec* status_out_dev, void* cuda_stream);

/* ---- (e) host scheduler: Algorithm 1 driving the calls above ---------------------------------- */

/*
 * AsyncLane active-lane decoding (Alg.1) of ONE sequence, as host control flow around the
 * device calls: per iteration the active lanes A_t (Eq.10) are packed into lane descriptors,
 * the model is called once for all of them (Eq.11), al_confidence_select applies the transfer rule
 * (refine lanes suppress EOS; one token per lane is forced so that a lane's budget is finite, reading
 * C4), al_lane_status returns the per-lane integers, and the host applies the fork operator (Eq.6),
 * completion / successor spawning with cascading termination (Eq.9, Alg.1 lines 10-17) and the
 * periodic compact refresh (Eq.12).  COLLECTDFS reconstructs the output.
 * Readings (C18-C21): a lane forks when 0 < p_l < b_l, n_filled / b_l >= rho_min, t_l >= t_min
 * and it still holds a MASK; the refine child covers [s, s + p) with a fresh clock, the continuation starts
 * at s + p with min(B, L - (s + p)) tokens; a lane is completed when it holds no MASK or after max_lane_steps
 * steps; a completed unforked generate lane spawns a successor at s + v_l unless v_l = 0 or s + v_l >= L;
 * generate lanes get a lookahead window of min(W, L - (s + b)) rows; all lanes of the sequence share the
 * cache rows (group 0, kv_base_row 0) and see prefix_len = P + s of them (reading C1).
 * The model is a callback: it receives the iteration's lanes (host copies), each lane's local step, the
 * packed input rows tokens_dev [n_rows] (device), row_pos_dev [2][n_rows] (device: the rows' positions in
 * generation coordinates, then the rows' lane-local steps), and writes fp32 logits [n_rows][vocab] (device)
 * on the given stream; it returns 0 on success.  al_stub_model_fn is a table-driven stand-in for tests and benchmarks (there are no
 * weights here): logits[row][v] = base[pos][v] + gain * (step + 1) * (v == target[pos]).
 * This entry allocates its own device and pinned buffers, synchronises once per iteration (the scheduler
 * reads 32 bytes per lane and the transferred tokens back) and frees everything before it returns.
 */
typedef struct {
  int32_t prompt_len, gen_len, block_size, lookahead;      /* P, L, B, W                                  */
  int32_t vocab, mask_id, eos_id;
  float tau, tau_future, rho_min;                          /* transfer / draft thresholds, Eq.5 fill ratio */
  int32_t t_min, max_lane_steps, max_iterations;           /* Eq.5 t_min; denoising budget per lane; total */
  int32_t refresh_period, refresh_margin;                  /* iterations between refreshes (0: never); m   */
  const int32_t* delimiter_ids;    int32_t n_delimiters;   /* HOST arrays: D_task                         */
  const int32_t* no_fork_prev_ids; int32_t n_no_fork_prev; /*              ValidBoundary exclusion        */
} al_sched_config;

typedef struct {             /* one node of the lane tree T_lane (host) */
  int32_t role;              /* 0 generate, 1 refine                                                       */
  int32_t start, len, steps; /* s_l, b_l, t_l                                                              */
  int32_t parent, ref_child, gen_child, successor;   /* node indices, -1 = none                           */
  int32_t state;             /* 0 active, 1 completed, 2 forked                                            */
  int32_t valid_prefix, split_point, n_masked;       /* as of the lane's last update                      */
} al_sched_lane;

typedef struct {
  int32_t iterations, model_calls, lane_forwards, forks, successors, refreshes, stopped_frontiers;
  int32_t rows_forwarded, tokens_committed, tokens_drafted, refreshed_rows_last, reserved;
} al_sched_stats;

typedef int (*al_model_fn)(void* user, const al_lane_desc* lanes_host, const int32_t* lane_steps_host,
                           int32_t n_lanes, int32_t n_rows, const int32_t* row_pos_dev,
                           const int32_t* tokens_dev, float* logits_dev, void* cuda_stream);

typedef struct {             /* user data of al_stub_model_fn; the tables live in DEVICE memory */
  const float* base_dev;     /* [gen_len][vocab]                                                           */
  const int32_t* target_dev; /* [gen_len]                                                                  */
  float gain;
  int32_t vocab;
} al_stub_model;
int al_stub_model_fn(void* user, const al_lane_desc* lanes_host, const int32_t* lane_steps_host,
                     int32_t n_lanes, int32_t n_rows, const int32_t* row_pos_dev, const int32_t* tokens_dev,
                     float* logits_dev, void* cuda_stream);

typedef struct {             /* optional device state the scheduler drives besides the logits (may be NULL) */
  al_attn_shape shape;       /* cache_rows >= P + L                                                        */
  void* k_cache; void* v_cache;            /* [H_kv][cache_rows][d]: refreshed rows are written here      */
  const void* k_src; const void* v_src;    /* [P + L][H_kv][d]: recomputed prefix states (Eq.12 source)   */
  const void* q; const void* k_new; const void* v_new;   /* [max_rows][H][d] lane inputs of the stub layer */
  void* out;                               /* [max_rows][H_q][d]; NULL q => no attention is run           */
  int32_t max_rows;
} al_sched_device_state;

/*
 * prompt_host [P]; x_host [P + L] receives the final global token state; output_host [L] the collected
 * sequence (n_output tokens); tree_out [max_tree] the lane tree (n_tree nodes; node 0 is the root).
 * Returns AL_ERR_UNSUPPORTED when the tree outgrows max_tree, AL_ERR_CUDA when the model callback fails.
 */
al_status al_scheduler_run(al_handle* handle, const al_sched_config* config, al_model_fn model,
                           void* model_user, const al_sched_device_state* device_state_or_null,
                           const int32_t* prompt_host, int32_t* x_host, int32_t* output_host,
                           int32_t* n_output, al_sched_lane* tree_out, int32_t max_tree, int32_t* n_tree,
                           al_sched_stats* stats_out, void* cuda_stream);

/* ---- whole step from HOST buffers (end-to-end entry) ------------------------------------------ */

/*
 * One lane-batched denoising step (all n_layers layers) whose per-step inputs
 * and results live in HOST memory (pinned for true asynchrony): the call validates all three parts
 * (on error nothing has been enqueued), then enqueues, on `cuda_stream`, the host->device copies of
 * the inputs into `arena_dev`, al_lane_plan once and al_lane_attention_planned per layer, the
 * layer-batched al_kv_refresh and al_confidence_select on the device copies, then the device->host
 * copies of the results.  It does not synchronise: the caller synchronises the stream before reading
 * the outputs or reusing the host inputs.  The KV cache is persistent device state (PAPER.md L70:
 * kappa_l is carried between iterations) and is passed as device pointers, layers
 * `cache_layer_stride` elements apart; attention reads it before this step's refresh writes it.
 * Every pointer inside al_host_step is a HOST pointer owned by the caller; L = max(n_layers, 1).
 */
typedef struct {
  const void* q;            /* [L][T][H_q][d]                               */
  const void* k_new;        /* [L][T][H_kv][d]                              */
  const void* v_new;        /* [L][T][H_kv][d]                              */
  const al_lane_desc* lanes;/* [n_lanes]                                    */
  int32_t n_lanes, total_q_rows, max_prefix_len;
  const void* k_src;        /* [L][n_pos][H_kv][d] recomputed rows (Eq.12)  */
  const void* v_src;
  const int32_t* pos;       /* [n_pos] strictly increasing                  */
  int32_t n_pos, refresh_base_row;
  const void* logits;       /* [n_rows][vocab], dtype = shape->dtype        */
  int32_t n_rows, vocab;
  const int32_t* tokens_in; /* [n_rows]                                     */
  int32_t mask_id, eos_id;
  float threshold;
  int32_t select_flags;     /* AL_SELECT_*                                  */
  void* out;                /* [L][T][H_q][d]   result, host                */
  float* conf;              /* [n_rows]                                     */
  int32_t* argmax;          /* [n_rows]                                     */
  uint8_t* commit;          /* [n_rows]                                     */
  int32_t* tokens_out;      /* [n_rows]                                     */
  int32_t n_layers;         /* layers of the model call; 0 is read as 1     */
  int32_t reserved;         /* must be 0                                    */
  int64_t cache_layer_stride; /* elements between layers of k/v_cache_dev   */
} al_host_step;

/* Bytes of device scratch al_lane_step_host needs for these sizes (0 on invalid arguments). */
size_t al_lane_step_host_arena_bytes(const al_attn_shape* shape, const al_host_step* step);
al_status al_lane_step_host(al_handle* handle, const al_attn_shape* shape, const al_host_step* step,
                            void* k_cache_dev, void* v_cache_dev, void* arena_dev,
                            size_t arena_bytes, void* cuda_stream);
/* Bytes copied host->device / device->host by one al_lane_step_host call with these sizes. */
void al_lane_step_host_traffic(const al_attn_shape* shape, const al_host_step* step,
                               uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* Number of kernel launches this handle has enqueued so far (bench accounting; a captured graph
 * counts its launches once, at capture). */
uint64_t al_launch_count(const al_handle* handle);

/* ---- debug / self-test (synchronising; never on the hot path) --------------------------------- */

/* Copies the descriptors to the host and checks the preconditions listed above.  Synchronises. */
al_status al_validate_lanes(al_handle* handle, const al_attn_shape* shape,
                            const al_lane_desc* lanes_dev, int32_t n_lanes, int32_t total_q_rows);
/* Copies the refresh positions to the host and checks al_kv_refresh's preconditions (Eq.12
 * rewrites each refreshed position once): pos strictly increasing -- hence unique -- and every
 * kv_base_row + pos[r] inside [0, cache_rows).  Synchronises. */
al_status al_validate_refresh(al_handle* handle, const al_attn_shape* shape, const int32_t* pos_dev,
                              int32_t n_pos, int32_t kv_base_row);

/*
 * tcgen05 encoding self-test: one 128x128x128 bf16 tile pipeline through the same TMA maps, shared
 * memory descriptors, instruction descriptors and TMEM paths as the attention kernel:
 *   s_out[128][128] (f32) = A . B^T                (A, B: [128][128] bf16, K-major)
 *   o_out[128][128] (f32) = bf16(s_out * p_scale) . V   (V: [128 keys][128] bf16, P fed from TMEM)
 * Synchronises.  All pointers are device pointers.
 */
al_status al_selftest_umma(al_handle* handle, const void* a_bf16, const void* b_bf16,
                           const void* v_bf16, float p_scale, float* s_out, float* o_out,
                           void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* ASYNCLANE_H_ */
