// k3_mlp_fp32.cuh -- K3 (FP32 FFMA path): per-element MLP 384->160->128->96->1 with
// CELU(0.1), forward and input-gradient backward, fused per 64-row tile
// (O5; backward = PAPER.md:67 "forces by backprop", weight gradients
// are never needed).
//
// Rows are atoms of ONE element (element blocks are padded to ROW_PAD rows), so
// a tile is a dense [64 x K] x [K x N] contraction chain -- a grouped GEMM over
// the four element blocks.  Activations stay in shared memory, k-major
// (XT[k][m], stride 68 floats) so a warp's 8-row A fragment is two broadcast
// LDS.128; weights stream from L2 through a cp.async double buffer, laid out
// [k][n] for every GEMM (forward uses transposed copies made by pfc_create).
// Thread tile: 8 rows (warp w -> rows 8w..8w+7) x N/32 columns (lane + 32c).
// This path is kept as the in-tolerance FP32 reference for the tensor-core path.
#pragma once
#include "pfc_common.cuh"

namespace pfc {

constexpr int MLP_TM = 64;
constexpr int MLP_THREADS = 256;
constexpr int MLP_KC = 16;
constexpr int MLP_LDT = MLP_TM + 4;      // 68: k-major activation stride
constexpr int MLP_BS_FLOATS = MLP_KC * D1;   // one staging buffer (widest N = 160)
constexpr size_t MLP_FP32_SMEM =
    sizeof(float) * ((size_t)(D0 + D1 + D2 + D3) * MLP_LDT + 2 * MLP_BS_FLOATS);   // 229,376 B

struct MlpWeights {          // device pointers, one set per element
  const float *W1t, *b1, *W2t, *b2, *W3t, *b3, *W4, *b4;   // forward: [k][n]
  const float *W1, *W2, *W3;                               // backward: original [out][in]
};
struct MlpParams {
  MlpWeights w[NSPEC];
  int row_start[NSPEC + 1];  // element block boundaries in padded row order
};

__device__ __forceinline__ float celu_f(float x) {
  return x > 0.0f ? x : CELU_ALPHA * (expf(x * (1.0f / CELU_ALPHA)) - 1.0f);
}
// CELU'(z) recovered from h = CELU(z): 1 for h > 0, exp(z/alpha) = h/alpha + 1 otherwise
__device__ __forceinline__ float dcelu_from_h(float h) {
  return h > 0.0f ? 1.0f : fmaf(h, 1.0f / CELU_ALPHA, 1.0f);
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// acc[r][c] = sum_k AT[k][8w + r] * B[k][n0 + lane + 32c],  k < K
template <int K, int N>
__device__ __forceinline__ void mlp_gemm(const float* __restrict__ AT, const float* __restrict__ Bg,
                                         int ldb, float* __restrict__ Bs, float (&acc)[8][N / 32]) {
  constexpr int NT = N / 32;
  constexpr int NCH = K / MLP_KC;
  constexpr int V4 = MLP_KC * N / 4;                     // float4s per chunk
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
  for (int r = 0; r < 8; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) acc[r][c] = 0.0f;
  auto stage = [&](int ch, int buf) {
    const float* src = Bg + (size_t)ch * MLP_KC * ldb;
    float* dst = Bs + buf * MLP_BS_FLOATS;
    for (int q = tid; q < V4; q += MLP_THREADS) {
      const int kk = q / (N / 4), n4 = q - kk * (N / 4);
      cp_async16(dst + kk * N + 4 * n4, src + (size_t)kk * ldb + 4 * n4);
    }
    cp_async_commit();
  };
  __syncthreads();                                       // previous users of Bs / writers of AT done
  stage(0, 0);
  for (int ch = 0; ch < NCH; ++ch) {
    if (ch + 1 < NCH) { stage(ch + 1, (ch + 1) & 1); cp_async_wait<1>(); }
    else cp_async_wait<0>();
    __syncthreads();
    const float* bs = Bs + (ch & 1) * MLP_BS_FLOATS + lane;
    const float* at = AT + (size_t)ch * MLP_KC * MLP_LDT + 8 * w;
#pragma unroll
    for (int kk = 0; kk < MLP_KC; ++kk) {
      const float4 a0 = *reinterpret_cast<const float4*>(at + kk * MLP_LDT);
      const float4 a1 = *reinterpret_cast<const float4*>(at + kk * MLP_LDT + 4);
      const float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      float b[NT];
#pragma unroll
      for (int c = 0; c < NT; ++c) b[c] = bs[kk * N + 32 * c];
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < NT; ++c) acc[r][c] = fmaf(a[r], b[c], acc[r][c]);
    }
    __syncthreads();
  }
}

// store an [8 x NT] thread tile k-major: HT[n][8w + r]
template <int NT>
__device__ __forceinline__ void store_tile_T(float* __restrict__ HT, const float (&v)[8][NT]) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int c = 0; c < NT; ++c) {
    float* p = HT + (size_t)(lane + 32 * c) * MLP_LDT + 8 * w;
    *reinterpret_cast<float4*>(p) = make_float4(v[0][c], v[1][c], v[2][c], v[3][c]);
    *reinterpret_cast<float4*>(p + 4) = make_float4(v[4][c], v[5][c], v[6][c], v[7][c]);
  }
}

__global__ void __launch_bounds__(MLP_THREADS, 1)
k3_mlp_fp32_kernel(const __grid_constant__ MlpParams P, const float* __restrict__ aev,
                   float* __restrict__ g, float* __restrict__ e_row) {
  extern __shared__ __align__(16) float smem[];
  float* XT = smem;
  float* H1T = XT + D0 * MLP_LDT;
  float* H2T = H1T + D1 * MLP_LDT;
  float* H3T = H2T + D2 * MLP_LDT;
  float* Bs = H3T + D3 * MLP_LDT;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int row0 = blockIdx.x * MLP_TM;
  int el = 0;
#pragma unroll
  for (int q = 1; q < NSPEC; ++q) el += (row0 >= P.row_start[q]);
  const MlpWeights W = P.w[el];

  // AEV tile -> XT (transposed): warp w loads rows 8w..8w+7, lanes along k
  for (int r = 0; r < 8; ++r) {
    const float* src = aev + (size_t)(row0 + 8 * w + r) * AEV_LEN;
#pragma unroll
    for (int q = 0; q < AEV_LEN / 32; ++q) XT[(size_t)(lane + 32 * q) * MLP_LDT + 8 * w + r] = src[lane + 32 * q];
  }
  // ---- forward ----
  {
    float acc[8][D1 / 32];
    mlp_gemm<D0, D1>(XT, W.W1t, D1, Bs, acc);
#pragma unroll
    for (int c = 0; c < D1 / 32; ++c) {
      const float bias = W.b1[lane + 32 * c];
#pragma unroll
      for (int r = 0; r < 8; ++r) acc[r][c] = celu_f(acc[r][c] + bias);
    }
    store_tile_T<D1 / 32>(H1T, acc);
  }
  {
    float acc[8][D2 / 32];
    mlp_gemm<D1, D2>(H1T, W.W2t, D2, Bs, acc);
#pragma unroll
    for (int c = 0; c < D2 / 32; ++c) {
      const float bias = W.b2[lane + 32 * c];
#pragma unroll
      for (int r = 0; r < 8; ++r) acc[r][c] = celu_f(acc[r][c] + bias);
    }
    store_tile_T<D2 / 32>(H2T, acc);
  }
  {
    float acc[8][D3 / 32];
    mlp_gemm<D2, D3>(H2T, W.W3t, D3, Bs, acc);
    float part[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int c = 0; c < D3 / 32; ++c) {
      const float bias = W.b3[lane + 32 * c], w4 = W.W4[lane + 32 * c];
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const float h = celu_f(acc[r][c] + bias);
        part[r] = fmaf(w4, h, part[r]);
        acc[r][c] = w4 * dcelu_from_h(h);               // delta3 = dE/dz3
      }
    }
    store_tile_T<D3 / 32>(H3T, acc);
    const float b4 = W.b4[0];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      const float s = warp_sum(part[r]);
      if (lane == 0) e_row[row0 + 8 * w + r] = s + b4;
    }
  }
  // ---- backward (input gradient only) ----
  {
    float acc[8][D2 / 32];
    mlp_gemm<D3, D2>(H3T, W.W3, D2, Bs, acc);
#pragma unroll
    for (int c = 0; c < D2 / 32; ++c) {
      const float* hp = H2T + (size_t)(lane + 32 * c) * MLP_LDT + 8 * w;
#pragma unroll
      for (int r = 0; r < 8; ++r) acc[r][c] *= dcelu_from_h(hp[r]);
    }
    store_tile_T<D2 / 32>(H2T, acc);                    // delta2 over h2 (own elements only)
  }
  {
    float acc[8][D1 / 32];
    mlp_gemm<D2, D1>(H2T, W.W2, D1, Bs, acc);
#pragma unroll
    for (int c = 0; c < D1 / 32; ++c) {
      const float* hp = H1T + (size_t)(lane + 32 * c) * MLP_LDT + 8 * w;
#pragma unroll
      for (int r = 0; r < 8; ++r) acc[r][c] *= dcelu_from_h(hp[r]);
    }
    store_tile_T<D1 / 32>(H1T, acc);                    // delta1
  }
#pragma unroll 1
  for (int n0 = 0; n0 < D0; n0 += 128) {
    float acc[8][4];
    mlp_gemm<D1, 128>(H1T, W.W1 + n0, D0, Bs, acc);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      float* dst = g + (size_t)(row0 + 8 * w + r) * AEV_LEN + n0 + lane;
#pragma unroll
      for (int c = 0; c < 4; ++c) dst[32 * c] = acc[r][c];
    }
  }
}

}  // namespace pfc
