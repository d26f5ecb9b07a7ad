// rotattn_probe_gemm8: a plain persistent tcgen05 8-bit GEMM, used to MEASURE the dense INT8 (and
// integer-valued E4M3) tensor rate on this GPU and to validate the descriptor / TMEM layouts the
// attention kernels rely on.  Not on the hot path.
#include <cstdio>
#include "tc_common.cuh"

namespace rotattn {

constexpr int GM = 128, GN = 256, GK = 128;       // CTA tile; GK bytes = one 128-byte swizzle row
constexpr int GSTAGES = 4;
constexpr int G_A_BYTES = GM * GK, G_B_BYTES = GN * GK;
constexpr int G_SMEM = GSTAGES * (G_A_BYTES + G_B_BYTES) + 1024 /*align*/ + 256 /*barriers*/;

template <MmaKind KIND>
__global__ void __launch_bounds__(256, 1)
gemm8_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, uint32_t* __restrict__ C,
             int M, int N, int K) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* sA = smem;
  uint8_t* sB = smem + GSTAGES * G_A_BYTES;
  uint64_t* bars = (uint64_t*)(smem + GSTAGES * (G_A_BYTES + G_B_BYTES));
  uint64_t* full = bars;                 // [GSTAGES]
  uint64_t* empty = bars + GSTAGES;      // [GSTAGES]
  uint64_t* tfull = bars + 2 * GSTAGES;  // [2]
  uint64_t* tempty = tfull + 2;          // [2]
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int i = 0; i < GSTAGES; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 128); }
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int tiles_n = N / GN, ntiles = (M / GM) * tiles_n, nkb = K / GK;
  constexpr uint32_t idesc = KIND == MmaKind::I8 ? umma_idesc(2, 1, 1, GM, GN) : umma_idesc(1, 0, 0, GM, GN);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA); tma_prefetch_desc(&tmB);
    int s = 0; uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const int m0 = (tile / tiles_n) * GM, n0 = (tile % tiles_n) * GN;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(&empty[s], ph ^ 1);
        mbar_arrive_expect_tx(&full[s], G_A_BYTES + G_B_BYTES);
        tma_load_3d(sA + s * G_A_BYTES, &tmA, &full[s], kb * GK, m0, 0);
        tma_load_3d(sB + s * G_B_BYTES, &tmB, &full[s], kb * GK, n0, 0);
        if (++s == GSTAGES) { s = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1 && lane == 0) {
    int s = 0; uint32_t ph = 0; int acc = 0; uint32_t aph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      mbar_wait(&tempty[acc], aph ^ 1);
      tc_fence_after();
      const uint32_t d = tmem_base + acc * GN;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(&full[s], ph);
        tc_fence_after();
        const uint64_t ad = umma_desc_k128(smem_u32(sA + s * G_A_BYTES));
        const uint64_t bd = umma_desc_k128(smem_u32(sB + s * G_B_BYTES));
#pragma unroll
        for (int k = 0; k < GK / 32; ++k) mma_ss<KIND>(d, ad + 2 * k, bd + 2 * k, idesc, (kb | k) != 0);
        tc_commit(&empty[s]);
        if (++s == GSTAGES) { s = 0; ph ^= 1; }
      }
      tc_commit(&tfull[acc]);
      if (++acc == 2) { acc = 0; aph ^= 1; }
    }
  } else if (warp >= 4) {
    const int q = warp & 3;
    int acc = 0; uint32_t aph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const int m0 = (tile / tiles_n) * GM, n0 = (tile % tiles_n) * GN;
      mbar_wait(&tfull[acc], aph);
      tc_fence_after();
      uint32_t* crow = C + (size_t)(m0 + q * 32 + lane) * N + n0;
#pragma unroll 1
      for (int c = 0; c < GN / 32; ++c) {
        uint32_t r[32];
        tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + acc * GN + c * 32, r);
        tmem_wait_ld();
#pragma unroll
        for (int j = 0; j < 8; ++j)
          *reinterpret_cast<uint4*>(crow + c * 32 + j * 4) = make_uint4(r[4 * j], r[4 * j + 1], r[4 * j + 2], r[4 * j + 3]);
      }
      tc_fence_before();
      mbar_arrive(&tempty[acc]);
      if (++acc == 2) { acc = 0; aph ^= 1; }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

// mode 2: one 128x128x128 tile, A (u8) staged through tensor memory, B (s8) via TMA; 128 threads.
__global__ void __launch_bounds__(128, 1)
gemm8_ts_kernel(const uint8_t* __restrict__ A, const __grid_constant__ CUtensorMap tmB, int32_t* __restrict__ C) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* sB = smem;
  uint64_t* bars = (uint64_t*)(smem + 128 * 128);
  uint32_t* tmem_slot = (uint32_t*)(bars + 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); fence_mbar_init(); }
  if (warp == 0) tmem_alloc(tmem_slot, 256);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t lane_off = (uint32_t)(warp * 32) << 16;
  if (threadIdx.x == 0) {
    mbar_arrive_expect_tx(&bars[0], 128 * 128);
    tma_load_3d(sB, &tmB, &bars[0], 0, 0, 0);
  }
  // row r = threadIdx.x of A: 128 bytes = 32 words -> TMEM columns [128, 160)
  {
    uint32_t w[32];
    const uint4* src = reinterpret_cast<const uint4*>(A + (size_t)threadIdx.x * 128);
#pragma unroll
    for (int j = 0; j < 8; ++j) { uint4 v = src[j]; w[4 * j] = v.x; w[4 * j + 1] = v.y; w[4 * j + 2] = v.z; w[4 * j + 3] = v.w; }
    tmem_st32(tmem_base + lane_off + 128, w);
    tmem_wait_st();
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) {
    tc_fence_after();
    mbar_wait(&bars[0], 0);
    tc_fence_after();
    constexpr uint32_t idesc = umma_idesc(2, 0 /*A u8*/, 1 /*B s8*/, 128, 128);
    const uint64_t bd = umma_desc_k128(smem_u32(sB));
#pragma unroll
    for (int k = 0; k < 4; ++k) mma_ts<MmaKind::I8>(tmem_base, tmem_base + 128 + 8 * k, bd + 2 * k, idesc, k != 0);
    tc_commit(&bars[1]);
  }
  mbar_wait(&bars[1], 0);
  tc_fence_after();
  int32_t* crow = C + (size_t)threadIdx.x * 128;
#pragma unroll 1
  for (int c = 0; c < 4; ++c) {
    uint32_t r[32];
    tmem_ld32(tmem_base + lane_off + c * 32, r);
    tmem_wait_ld();
#pragma unroll
    for (int j = 0; j < 32; ++j) crow[c * 32 + j] = (int32_t)r[j];
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, 256);
}

}  // namespace rotattn

using namespace rotattn;

extern "C" int rotattn_probe_gemm8(int32_t M, int32_t N, int32_t K, const void* A, const void* B, void* C,
                                   int32_t mode, void* stream) {
  if (!A || !B || !C || mode < 0 || mode > 2) return ROTATTN_ERR_INVALID_ARG;
  if (M < GM || N < 128 || K < GK || M % GM || K % GK) return ROTATTN_ERR_INVALID_ARG;
  int st = check_device_sm100();
  if (st != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  CUtensorMap tmA, tmB;
  if (mode == 2) {
    if (M != 128 || N != 128 || K != 128) return ROTATTN_ERR_INVALID_ARG;
    if ((st = make_tmap_3d(&tmB, B, 1, K, N, 1, K, (uint64_t)N * K, 128, 128)) != ROTATTN_OK) return st;
    const int smem = 128 * 128 + 1024 + 64;
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(gemm8_ts_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    gemm8_ts_kernel<<<1, 128, smem, cs>>>((const uint8_t*)A, tmB, (int32_t*)C);
    ROTATTN_CUDA_TRY(cudaGetLastError());
    return ROTATTN_OK;
  }
  if (N % GN) return ROTATTN_ERR_INVALID_ARG;
  if ((st = make_tmap_3d(&tmA, A, 1, K, M, 1, K, (uint64_t)M * K, 128, GM)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tmB, B, 1, K, N, 1, K, (uint64_t)N * K, 128, GN)) != ROTATTN_OK) return st;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ntiles = (M / GM) * (N / GN);
  const int grid = ntiles < sms ? ntiles : sms;
  if (mode == 0) {
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(gemm8_kernel<MmaKind::I8>, cudaFuncAttributeMaxDynamicSharedMemorySize, G_SMEM));
    gemm8_kernel<MmaKind::I8><<<grid, 256, G_SMEM, cs>>>(tmA, tmB, (uint32_t*)C, M, N, K);
  } else {
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(gemm8_kernel<MmaKind::F8F6F4>, cudaFuncAttributeMaxDynamicSharedMemorySize, G_SMEM));
    gemm8_kernel<MmaKind::F8F6F4><<<grid, 256, G_SMEM, cs>>>(tmA, tmB, (uint32_t*)C, M, N, K);
  }
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}
