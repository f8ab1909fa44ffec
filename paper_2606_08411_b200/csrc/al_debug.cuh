// Debug instrumentation of the attention kernel: clock64 stamps per CTA / step / warp and a recording
// variant of the barrier time-out.  Everything here is compiled only with -DAL_ATTN_TRACE
// (AL_NVCC_EXTRA=-DAL_ATTN_TRACE python -m paper_2606_08411_b200.build --force); a release build sees
// empty macros and none of the globals or the al_debug_* exports.
#pragma once

#ifdef AL_ATTN_TRACE
// per-CTA clock64 stamps of the first piece (slot 15 = globaltimer at entry)
__device__ unsigned long long g_trace[256 * 16];
#define TRACE(i) do { if (g_trace[blockIdx.x * 16 + (i)] == 0) g_trace[blockIdx.x * 16 + (i)] = clock64(); } while (0)
// CTA 0 only: per step (first 32 of the CTA) stamps of kind k: 0 QK_A issued, 1 S seen by stream A, 2 P_A ready, 3 PV_A issued
__device__ unsigned long long g_trace_tile[16 * 32];
#define TRACE_TILE(k, i) do { if (blockIdx.x == 0 && (i) < 32) g_trace_tile[(k) * 32 + (i)] = clock64(); } while (0)
// CTA 0, step 4 of each stream: per warp (8 softmax warps) stamps 0 S seen, 1 S in registers, 2 max done, 3 P stored, 4 arrived
__device__ unsigned long long g_trace_warp[8 * 8];
#define TRACE_W(k) do { if (blockIdx.x == 0 && cnt == 4 && lane == 0) g_trace_warp[(warp - 4) * 8 + (k)] = clock64(); } while (0)
__device__ unsigned long long g_trace_epi[16];
#define TRACE_E(k) do { if (blockIdx.x == 0 && warp == 4 && lane == 0 && g_trace_epi[k] == 0) g_trace_epi[k] = clock64(); } while (0)
#define TRACE_M(k) do { if (blockIdx.x == 12 && tid128 == 0 && b == 0 && g_trace_epi[k] == 0) g_trace_epi[k] = clock64(); } while (0)
#define TRACE_RESET()                                                                                          \
  do {                                                                                                         \
    if (threadIdx.x == 0) {                                                                                    \
      if (blockIdx.x == 0 || blockIdx.x == 12)                                                                 \
        for (int i_ = (blockIdx.x ? 11 : 0); i_ < (blockIdx.x ? 16 : 11); ++i_) g_trace_epi[i_] = 0;           \
      for (int i_ = 0; i_ < 16; ++i_) g_trace[blockIdx.x * 16 + i_] = 0;                                       \
      unsigned long long gt_;                                                                                  \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_));                                                  \
      g_trace[blockIdx.x * 16 + 15] = gt_;                                                                     \
      g_trace[blockIdx.x * 16 + 0] = clock64();                                                                \
    }                                                                                                          \
  } while (0)
// plan kernel: clock64 stamps after each phase (thread 0)
__device__ unsigned long long g_trace_plan[32];
#define TRACE_P(i) do { if (threadIdx.x == 0) g_trace_plan[i] = clock64(); } while (0)
extern "C" int al_debug_plan_trace(unsigned long long* host_out) {        // [32]
  return (int)cudaMemcpyFromSymbol(host_out, g_trace_plan, sizeof(g_trace_plan));
}
extern "C" int al_debug_attn_trace(unsigned long long* host_out) {        // [256 * 16]
  return (int)cudaMemcpyFromSymbol(host_out, g_trace, sizeof(g_trace));
}
extern "C" int al_debug_attn_trace_epi(unsigned long long* host_out) {    // [16]
  return (int)cudaMemcpyFromSymbol(host_out, g_trace_epi, sizeof(g_trace_epi));
}
extern "C" int al_debug_attn_trace_warp(unsigned long long* host_out) {   // [8 * 8]
  return (int)cudaMemcpyFromSymbol(host_out, g_trace_warp, sizeof(g_trace_warp));
}
extern "C" int al_debug_attn_trace_tile(unsigned long long* host_out) {   // [16 * 32]
  return (int)cudaMemcpyFromSymbol(host_out, g_trace_tile, sizeof(g_trace_tile));
}
#else
#define TRACE(i) do { } while (0)
#define TRACE_TILE(k, i) do { } while (0)
#define TRACE_W(k) do { } while (0)
#define TRACE_E(k) do { } while (0)
#define TRACE_M(k) do { } while (0)
#define TRACE_RESET() do { } while (0)
#define TRACE_P(i) do { } while (0)
#endif
