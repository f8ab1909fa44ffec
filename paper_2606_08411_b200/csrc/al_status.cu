// al_lane_status -- the per-lane integers the host scheduler needs from one iteration, and the lookahead
// draft rule (Eq.8, Eq.5, Eq.9, Eq.4; Alg.1 L127-162 consumes them).
//
// K4  lane_status_kernel: one warp per lane, one launch.  A lane's rows are u_l = [z_l ; lookahead window]
//     (Eq.2): the first b = q_len - w rows are the lane state, the last w rows the window (w in flags bits
//     8..23).  The warp first decides the window rows by Eq.8 (drafted iff [MASK], q >= tau_future, greedy token
//     not EOS -- whatever the transfer rule wrote for them), then walks z_l in chunks of 32 rows: ballots give the
//     counts, the first MASK-or-EOS position (v_l) and the last valid delimiter (p_l).  Integer work on a few
//     hundred bytes per lane: latency-bound, it rides behind the confidence kernel with a programmatic
//     dependent launch, and its output (32 bytes per lane) is the ONE device-to-host copy of an iteration.
#include "al_internal.h"

namespace {

constexpr int kThreads = 128;

__device__ __forceinline__ bool in_set(int x, const int32_t* __restrict__ set, int n) {
  bool hit = false;
  for (int d = 0; d < n; ++d) hit |= (x == __ldg(set + d));
  return hit;
}

__global__ void __launch_bounds__(kThreads)
lane_status_kernel(const al_lane_desc* __restrict__ lanes, int n_lanes, int n_rows, const int32_t* __restrict__ tokens_in,
                   const float* __restrict__ conf, const int32_t* __restrict__ argmax, int mask_id, int eos_id,
                   float tau_future, const int32_t* __restrict__ delimiters, int n_delimiters,
                   const int32_t* __restrict__ no_fork_prev, int n_no_fork_prev, uint8_t* __restrict__ commit_io,
                   int32_t* __restrict__ tokens_io, al_lane_status_rec* __restrict__ status) {
  // programmatic dependent launch: conf / argmax / tokens of the select kernel are visible after the wait
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int lane = threadIdx.x & 31;
  const int l = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  if (l >= n_lanes) return;
  const int q_start = lanes[l].q_start, q_len = lanes[l].q_len;
  const int w = min(q_len, AL_LANE_LOOKAHEAD(lanes[l].flags));
  const int b = q_len - w;

  // Eq.8: the lookahead window
  int n_drafts = 0;
  for (int i = b + lane; i < q_len; i += 32) {
    const int row = q_start + i;
    if (row < 0 || row >= n_rows) continue;
    const int tin = tokens_in[row], am = argmax[row];
    const bool c = tin == mask_id && conf[row] >= tau_future && am != eos_id;
    commit_io[row] = c ? 1 : 0;
    tokens_io[row] = c ? am : tin;
    n_drafts += c ? 1 : 0;
  }
  // the lane state z_l after the transfer
  int n_filled = 0, n_committed = 0, v = b, p = 0;
  for (int i0 = 0; i0 < b; i0 += 32) {
    const int i = i0 + lane;
    const bool in = i < b;
    const int row = q_start + i;
    const int z = in ? tokens_io[row] : mask_id;
    const int zprev = (in && i > 0) ? tokens_io[row - 1] : mask_id;
    n_filled += (in && z != mask_id) ? 1 : 0;
    n_committed += (in && commit_io[row]) ? 1 : 0;
    const unsigned stop = __ballot_sync(0xffffffffu, in && (z == mask_id || z == eos_id));
    if (stop && v == b) v = i0 + __ffs(stop) - 1;            // the first chunk that holds one decides
    const bool delim = in && in_set(z, delimiters, n_delimiters) &&
                       !(i > 0 && in_set(zprev, no_fork_prev, n_no_fork_prev));
    const unsigned dm = __ballot_sync(0xffffffffu, delim);
    if (dm) p = i0 + (32 - __clz(dm));                       // 1 + the last valid delimiter of the chunk
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    n_filled += __shfl_xor_sync(0xffffffffu, n_filled, off);
    n_committed += __shfl_xor_sync(0xffffffffu, n_committed, off);
    n_drafts += __shfl_xor_sync(0xffffffffu, n_drafts, off);
  }
  if (lane == 0) {
    al_lane_status_rec r;
    r.n_filled = n_filled; r.valid_prefix = v; r.split_point = p; r.n_committed = n_committed;
    r.n_drafts = n_drafts; r.n_masked = b - n_filled; r.reserved[0] = r.reserved[1] = 0;
    status[l] = r;
  }
}

}  // namespace

extern "C" al_status al_lane_status(al_handle* h, const al_lane_desc* lanes, int32_t n_lanes, int32_t n_rows,
                                    const int32_t* tokens_in, const float* conf, const int32_t* argmax,
                                    int32_t mask_id, int32_t eos_id, float tau_future, const int32_t* delimiters,
                                    int32_t n_delimiters, const int32_t* no_fork_prev, int32_t n_no_fork_prev,
                                    uint8_t* commit_io, int32_t* tokens_io, al_lane_status_rec* status_out,
                                    void* stream) {
  const char* who = "al_lane_status";
  if (!h) AL_FAIL(AL_ERR_INVALID_ARG, "%s: handle is NULL", who);
  if (n_lanes < 0 || n_rows < 0 || n_delimiters < 0 || n_no_fork_prev < 0)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: negative size", who);
  if (n_lanes == 0) return AL_OK;
  const al_status st = al_check_device(h, who);
  if (st != AL_OK) return st;
  if (!lanes || !tokens_in || !conf || !argmax || !commit_io || !tokens_io || !status_out)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL pointer", who);
  if ((n_delimiters > 0 && !delimiters) || (n_no_fork_prev > 0 && !no_fork_prev))
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: NULL id list with a positive count", who);
  if (tokens_io == tokens_in)
    AL_FAIL(AL_ERR_INVALID_ARG, "%s: tokens_io must not alias tokens_in (Eq.8 reads the token BEFORE the transfer)", who);
  const int warps_per_block = kThreads / 32;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)((n_lanes + warps_per_block - 1) / warps_per_block));
  cfg.blockDim = dim3(kThreads);
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.wait in the kernel
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  AL_CUDA_OK(cudaLaunchKernelEx(&cfg, lane_status_kernel, lanes, (int)n_lanes, (int)n_rows, tokens_in, conf, argmax,
                                (int)mask_id, (int)eos_id, tau_future, delimiters, (int)n_delimiters, no_fork_prev,
                                (int)n_no_fork_prev, commit_io, tokens_io, status_out));
  h->launches++;
  return AL_OK;
}
