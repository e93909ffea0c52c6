// tc_probe.cuh -- pfc_tc_chain_probe (include/pfc_debug.h): one accumulator chain of tcgen05.mma kind::f16
// instructions on operands given by the caller, raw fp32 accumulator back.  It exists so that a test can
// MEASURE how the tensor core's accumulate step rounds (toward zero, once per
// instruction) with sums whose exact value the test computes itself -- the hardware fact the truncation
// compensation of k3_mlp_tc.cuh rests on -- instead of inferring it from the MLP's errors.
//
// D[128 x 64] = sum over n_mma instructions of A_c[128 x 16] B_c[64 x 16]^T, instruction i taking the 16-k
// slice (i mod n_slices) of the caller's operands A[128][16 n_slices], B[64][16 n_slices] (fp32 values that
// are exactly representable in fp16; both operands K-major SWIZZLE_64B in shared memory, exactly as in K3).
#pragma once
#include <cuda_fp16.h>

#include "k3_mlp_tc.cuh"

namespace pfc {

constexpr int TCP_M = 128, TCP_N = 64, TCP_MAX_SLICES = 16;   // slices of 16 k; two slices per 32-k chunk

__global__ void __launch_bounds__(128, 1)
tc_chain_probe_kernel(const float* __restrict__ A, const float* __restrict__ B, int n_slices, int n_mma,
                      float* __restrict__ D) {
  extern __shared__ uint8_t tcp_raw[];
  uint8_t* base = tcp_raw + ((1024u - (tc::smem_u32(tcp_raw) & 1023u)) & 1023u);
  const int n_chunks = (n_slices + 1) / 2;
  uint8_t* sA = base;                                   // n_chunks x [128 x 32] fp16
  uint8_t* sB = sA + (size_t)n_chunks * TCP_M * 64;     // n_chunks x [64 x 32] fp16
  __shared__ uint64_t done;
  __shared__ uint32_t tmem_base;
  const int tid = threadIdx.x, warp = tid >> 5;
  const int K = 16 * n_slices;
  for (int q = tid; q < TCP_M * 32 * n_chunks; q += 128) {
    const int ch = q / (TCP_M * 32), r = (q / 32) % TCP_M, kk = q % 32, k = 32 * ch + kk;
    const __half v = __float2half_rn(k < K ? A[(size_t)r * K + k] : 0.0f);
    *reinterpret_cast<__half*>(sA + (size_t)ch * TCP_M * 64 + tc_sw64_off(r, kk)) = v;
  }
  for (int q = tid; q < TCP_N * 32 * n_chunks; q += 128) {
    const int ch = q / (TCP_N * 32), r = (q / 32) % TCP_N, kk = q % 32, k = 32 * ch + kk;
    const __half v = __float2half_rn(k < K ? B[(size_t)r * K + k] : 0.0f);
    *reinterpret_cast<__half*>(sB + (size_t)ch * TCP_N * 64 + tc_sw64_off(r, kk)) = v;
  }
  if (tid == 0) { tc::mbar_init(&done, 1); tc::mbar_fence_init(); }
  if (warp == 0) tc::tmem_alloc<64>(&tmem_base);
  tc::fence_proxy_async_smem();
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tb = tmem_base;
  if (tid == 0) {
    const uint32_t idesc = tc_idesc_f16(TCP_M, TCP_N);
    for (int i = 0; i < n_mma; ++i) {
      const int sl = i % n_slices, ch = sl >> 1, half = sl & 1;
      const uint64_t da = tc_desc_sw64(tc::smem_u32(sA + (size_t)ch * TCP_M * 64) + 32 * half);
      const uint64_t db = tc_desc_sw64(tc::smem_u32(sB + (size_t)ch * TCP_N * 64) + 32 * half);
      tc_mma_f16(tb, da, db, idesc, i == 0 ? 0u : 1u);
    }
    tc::mma_commit(&done);
  }
  tc::mbar_wait(&done, 0);
  tc::tc_fence_after();
  const int r = tid;                                    // warp w reads TMEM lanes 32 w .. 32 w + 31
#pragma unroll 1
  for (int c = 0; c < TCP_N / 16; ++c) {
    float v[16];
    tc::tmem_ld16(tb + ((uint32_t)(32 * warp) << 16) + 16 * c, v);
    tc::tmem_ld_wait();
#pragma unroll
    for (int k = 0; k < 16; ++k) D[(size_t)r * TCP_N + 16 * c + k] = v[k];
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<64>(tb);
}

}  // namespace pfc
