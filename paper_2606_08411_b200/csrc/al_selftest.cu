// al_selftest_umma -- one 128x128x128 bf16 tile through exactly the encodings al_lane_attention's
// tcgen05 kernel relies on: SWIZZLE_128B TMA maps, K-major smem descriptors (A, B of S = A.B^T),
// fp32 accumulator read-back (tcgen05.ld 32x32b), bf16 P written to TMEM (tcgen05.st) and used as
// the A operand of a TS-form MMA against an MN-major smem operand V (O = P.V).
// Debug entry: synchronises.  AL_SELFTEST_VARIANT=1 issues P.V as two N=64 MMAs (one per 64-column
// half of V) instead of one N=128 MMA with a leading-byte-offset between the halves.
#include <cstdlib>

#include "al_internal.h"
#include "al_ptx.cuh"

using namespace alptx;

namespace {

constexpr int kTile = 128;
constexpr int kHalfBytes = kTile * 64 * 2;   // [128 rows][64 bf16] = 16 KB, one swizzle-atom column

struct SelfSmem {
  alignas(1024) uint8_t a[2][kHalfBytes];
  alignas(1024) uint8_t b[2][kHalfBytes];
  alignas(1024) uint8_t v[2][kHalfBytes];
  uint64_t bar_load, bar_s, bar_o;
  uint32_t tmem_base;
};

__global__ void __launch_bounds__(128, 1)
selftest_umma_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                     const __grid_constant__ CUtensorMap map_v, float p_scale, float* __restrict__ s_out,
                     float* __restrict__ o_out, int variant) {
  extern __shared__ uint8_t smem_raw[];
  SelfSmem& sm = *reinterpret_cast<SelfSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int warp = threadIdx.x >> 5;

  if (threadIdx.x == 0) {
    mbar_init(&sm.bar_load, 1);
    mbar_init(&sm.bar_s, 1);
    mbar_init(&sm.bar_o, 1);
    fence_barrier_init();
  }
  if (warp == 0) tmem_alloc<512>(&sm.tmem_base);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  const uint32_t t_s = tmem, t_p = tmem + 128, t_o = tmem + 256;

  if (threadIdx.x == 0) {
    mbar_arrive_expect_tx(&sm.bar_load, 6 * kHalfBytes);
    for (int h = 0; h < 2; ++h) {
      tma_load_2d(sm.a[h], &map_a, &sm.bar_load, h * 64, 0);
      tma_load_2d(sm.b[h], &map_b, &sm.bar_load, h * 64, 0);
      tma_load_2d(sm.v[h], &map_v, &sm.bar_load, h * 64, 0);
    }
    mbar_wait(&sm.bar_load, 0);
    tc_fence_after();
    // S = A . B^T : both operands K-major; K = 128 = 2 halves x 4 steps of 16 elements (32 bytes)
    const uint32_t idesc = make_idesc_bf16(128, 128, 0, 0);
    for (int h = 0; h < 2; ++h)
      for (int k = 0; k < 4; ++k) {
        const uint64_t da = make_desc_sw128(smem_u32(sm.a[h]) + k * 32, 16, 1024);
        const uint64_t db = make_desc_sw128(smem_u32(sm.b[h]) + k * 32, 16, 1024);
        mma_ss(t_s, da, db, idesc, (h | k) ? 1u : 0u);
      }
    mma_commit(&sm.bar_s);
  }
  __syncwarp();
  mbar_wait(&sm.bar_s, 0);
  tc_fence_after();

  const int row = threadIdx.x;                       // warp w reads TMEM lanes 32w..32w+31
  const uint32_t lane_addr = (uint32_t)(warp * 32) << 16;
  for (int c = 0; c < 4; ++c) {
    uint32_t r[32];
    tmem_ld32(t_s + lane_addr + c * 32, r);
    tmem_wait_ld();
    uint32_t p[16];
#pragma unroll
    for (int i = 0; i < 32; ++i) s_out[row * kTile + c * 32 + i] = __uint_as_float(r[i]);
#pragma unroll
    for (int i = 0; i < 16; ++i)
      p[i] = pack_bf16x2(__uint_as_float(r[2 * i]) * p_scale, __uint_as_float(r[2 * i + 1]) * p_scale);
    tmem_st16(t_p + lane_addr + c * 16, p);          // P[row][k] bf16: column k/2, half k%2
  }
  tmem_wait_st();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (threadIdx.x == 0) {
    // O = P . V : A = P from TMEM (K-major by construction), B = V stored [key][d] => MN-major.
    // Per K step of 16 keys: A advances 8 TMEM columns, B advances 16 rows x 128 B = 2048 B.
    if (variant == 0) {
      const uint32_t idesc = make_idesc_bf16(128, 128, 0, 1);
      for (int k = 0; k < 8; ++k) {
        const uint64_t db = make_desc_sw128(smem_u32(sm.v[0]) + k * 2048, kHalfBytes, 1024);
        mma_ts(t_o, t_p + k * 8, db, idesc, k ? 1u : 0u);
      }
    } else {
      const uint32_t idesc = make_idesc_bf16(128, 64, 0, 1);
      for (int h = 0; h < 2; ++h)
        for (int k = 0; k < 8; ++k) {
          const uint64_t db = make_desc_sw128(smem_u32(sm.v[h]) + k * 2048, kHalfBytes, 1024);
          mma_ts(t_o + h * 64, t_p + k * 8, db, idesc, k ? 1u : 0u);
        }
    }
    mma_commit(&sm.bar_o);
  }
  __syncwarp();
  mbar_wait(&sm.bar_o, 0);
  tc_fence_after();
  for (int c = 0; c < 4; ++c) {
    uint32_t r[32];
    tmem_ld32(t_o + lane_addr + c * 32, r);
    tmem_wait_ld();
#pragma unroll
    for (int i = 0; i < 32; ++i) o_out[row * kTile + c * 32 + i] = __uint_as_float(r[i]);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

}  // namespace

// 2D row-major bf16 tensor [rows][cols] -> tensor map with a (64 x box_rows) box, 128-byte swizzle.
al_status al_make_map_2d(const al_handle* h, CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols,
                         uint32_t box_rows) {
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * 2};
  const cuuint32_t box[2] = {64, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = h->encode_tiled(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides,
                               box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) AL_FAIL(AL_ERR_CUDA, "cuTensorMapEncodeTiled(2d) failed: %d", (int)r);
  return AL_OK;
}

extern "C" al_status al_selftest_umma(al_handle* h, const void* a, const void* b, const void* v, float p_scale,
                                      float* s_out, float* o_out, void* stream) {
  if (!h || !a || !b || !v || !s_out || !o_out) AL_FAIL(AL_ERR_INVALID_ARG, "al_selftest_umma: NULL argument");
  CUtensorMap ma, mb, mv;
  al_status st;
  if ((st = al_make_map_2d(h, &ma, a, kTile, kTile, kTile)) != AL_OK) return st;
  if ((st = al_make_map_2d(h, &mb, b, kTile, kTile, kTile)) != AL_OK) return st;
  if ((st = al_make_map_2d(h, &mv, v, kTile, kTile, kTile)) != AL_OK) return st;
  const char* env = getenv("AL_SELFTEST_VARIANT");
  const int variant = env ? atoi(env) : 0;
  const size_t smem = sizeof(SelfSmem) + 1024;
  AL_CUDA_OK(cudaFuncSetAttribute(selftest_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  selftest_umma_kernel<<<1, 128, smem, cs>>>(ma, mb, mv, p_scale, s_out, o_out, variant);
  AL_CUDA_OK(cudaGetLastError());
  AL_CUDA_OK(cudaStreamSynchronize(cs));
  return AL_OK;
}
