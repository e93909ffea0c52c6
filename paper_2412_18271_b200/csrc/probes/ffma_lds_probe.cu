// ffma_lds_probe.cu -- what FFMA rate does a B200 SM sustain for an R x NT outer-product register
// tile, from registers only and fed by LDS.128 in K3's access pattern (16 row groups x 2 column
// groups per warp)?  No global traffic, no barriers, no epilogue: the practical ceiling that
// k3_mlp_fp32.cuh is measured against in DESIGN.md.  Output of one run: profiles/r1c_probes.md.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o ffma_lds_probe ffma_lds_probe.cu && ./ffma_lds_probe
#include <cstdio>
#include <cuda_runtime.h>
#include <cstdint>
// R x NT tile, per k4: R LDS.128 (A, rows stride LDA) + 4*NT/4 LDS.128 (B)
template <int R, int NT, bool WITH_LDS>
__global__ void __launch_bounds__(512, 1) k(float* out, int iters, int lda) {
  extern __shared__ __align__(16) float sm[];
  for (int i = threadIdx.x; i < 48 * 1024; i += blockDim.x) sm[i] = 1.0f + (i & 7) * 1e-3f;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const float* at = sm + (64 * (w >> 3) + (lane >> 1)) * lda;
  const float* bs = sm + 32 * 1024 + 4 * (2 * (w & 7) + (lane & 1));
  float acc[R][NT];
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) acc[r][c] = 0.f;
  float4 a[R]; float b[NT];
#pragma unroll
  for (int r = 0; r < R; ++r) a[r] = make_float4(1.f + r, 2.f, 3.f, 4.f);
#pragma unroll
  for (int c = 0; c < NT; ++c) b[c] = 1.f + c;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k4 = 0; k4 < 4; ++k4) {
      if (WITH_LDS) {
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = *reinterpret_cast<const float4*>(at + r * 16 * lda + 4 * k4 + 16 * (it & 3));
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (WITH_LDS) {
#pragma unroll
          for (int f = 0; f < NT / 4; ++f) {
            const float4 v = *reinterpret_cast<const float4*>(bs + ((4 * k4 + j) + 16 * (it & 3)) * 160 + 64 * f);
            b[4 * f] = v.x; b[4 * f + 1] = v.y; b[4 * f + 2] = v.z; b[4 * f + 3] = v.w;
          }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const float av = j == 0 ? a[r].x : j == 1 ? a[r].y : j == 2 ? a[r].z : a[r].w;
#pragma unroll
          for (int c = 0; c < NT; ++c) acc[r][c] = fmaf(av, b[c], acc[r][c]);
        }
      }
    }
  }
  float s = 0;
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) s += acc[r][c];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int R, int NT, bool L>
void run(const char* name, int threads, float* d) {
  cudaFuncSetAttribute(k<R, NT, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096;
  for (int rep = 0; rep < 2; ++rep) {
    cudaEventRecord(e0);
    k<R, NT, L><<<148, threads, 200 * 1024>>>(d, iters, 164);
    cudaEventRecord(e1); cudaDeviceSynchronize();
  }
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double ffma = (double)iters * 16 * R * NT * threads * 148;
  printf("%-28s threads %d: %.1f TFLOP/s (%.1f%% of 74.45) %s\n", name, threads, 2 * ffma / ms * 1e-9, 2 * ffma / ms * 1e-9 / 74.45 * 100,
         cudaGetErrorString(cudaGetLastError()));
}
int main() {
  float* d; cudaMalloc(&d, 148 * 1024 * 4);
  run<4, 8, false>("R4 NT8 regs only", 512, d);
  run<4, 8, false>("R4 NT8 regs only", 256, d);
  run<4, 8, true>("R4 NT8 + LDS", 512, d);
  run<4, 8, true>("R4 NT8 + LDS", 256, d);
  run<8, 8, true>("R8 NT8 + LDS", 256, d);
  run<8, 8, true>("R8 NT8 + LDS", 512, d);
  run<4, 4, true>("R4 NT4 + LDS", 512, d);
  run<2, 8, true>("R2 NT8 + LDS", 512, d);
  run<8, 4, true>("R8 NT4 + LDS", 512, d);
  run<8, 8, false>("R8 NT8 regs only", 256, d);
  return 0;
}
