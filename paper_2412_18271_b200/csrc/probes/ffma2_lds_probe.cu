// ffma2_lds_probe.cu -- the LDS-fed outer-product tile of ffma_lds_probe.cu with the packed
// fma.rn.f32x2 instruction (SASS FFMA2): accumulator pairs hold the (even k, odd k) partial sums, so
// the activation pair comes straight from the float4 along k and the weight pair from a k-pair
// interleaved layout.  Halves the FMA issue slots; whether that helps depends on threads per SM
// (profiles/r1c_probes.md): 70 % of nominal at 512 threads for the 2 x 8 tile (plain FFMA: 61 %),
// but 62 % at 768 threads -- K3's three co-resident 256-thread CTAs -- where plain FFMA also gives 62 %.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o ffma2_lds_probe ffma2_lds_probe.cu && ./ffma2_lds_probe
#include <cstdio>
#include <cuda_runtime.h>
__device__ __forceinline__ void ffma2(float2& acc, float2 a, float2 b) {
  unsigned long long ua = *reinterpret_cast<unsigned long long*>(&a), ub = *reinterpret_cast<unsigned long long*>(&b),
                     uc = *reinterpret_cast<unsigned long long*>(&acc), ud;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
  acc = *reinterpret_cast<float2*>(&ud);
}
template <int R, int NT, int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k(float* out, int iters, int lda) {
  extern __shared__ __align__(16) float sm[];
  for (int i = threadIdx.x; i < 48 * 1024; i += blockDim.x) sm[i] = 1.0f + (i & 7) * 1e-3f;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const float* at = sm + (64 * ((w >> 3) & 1) + (lane >> 1)) * lda;
  const float* bs = sm + 32 * 1024 + 4 * (2 * (w & 7) + (lane & 1));
  float2 acc[R][NT];
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) acc[r][c] = make_float2(0.f, 0.f);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k4 = 0; k4 < 4; ++k4) {
      float4 a[R];
#pragma unroll
      for (int r = 0; r < R; ++r) a[r] = *reinterpret_cast<const float4*>(at + r * 16 * lda + 4 * k4 + 16 * (it & 3));
#pragma unroll
      for (int j = 0; j < 2; ++j) {       // k pair
        float2 b[NT];
#pragma unroll
        for (int f = 0; f < NT / 2; ++f) {   // one LDS.128 = 2 columns x (k, k+1)
          const float4 v = *reinterpret_cast<const float4*>(bs + ((2 * k4 + j) + 8 * (it & 3)) * 320 + 128 * f);
          b[2 * f] = make_float2(v.x, v.y); b[2 * f + 1] = make_float2(v.z, v.w);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const float2 av = j == 0 ? make_float2(a[r].x, a[r].y) : make_float2(a[r].z, a[r].w);
#pragma unroll
          for (int c = 0; c < NT; ++c) ffma2(acc[r][c], av, b[c]);
        }
      }
    }
  }
  float s = 0;
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) s += acc[r][c].x + acc[r][c].y;
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int R, int NT, int THREADS>
void run(const char* name, float* d) {
  cudaFuncSetAttribute(k<R, NT, THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096;
  float ms;
  for (int rep = 0; rep < 2; ++rep) {
    cudaEventRecord(e0);
    k<R, NT, THREADS><<<148, THREADS, 200 * 1024>>>(d, iters, 164);
    cudaEventRecord(e1); cudaDeviceSynchronize();
  }
  cudaEventElapsedTime(&ms, e0, e1);
  double ffma = (double)iters * 16 * R * NT * THREADS * 148;
  printf("%-20s threads %4d: %.1f TFLOP/s (%.1f%% of 74.45) %s\n", name, THREADS, 2 * ffma / ms * 1e-9, 2 * ffma / ms * 1e-9 / 74.45 * 100,
         cudaGetErrorString(cudaGetLastError()));
}
int main() {
  float* d; cudaMalloc(&d, 148 * 1024 * 4);
  run<2, 8, 256>("R2 NT8 f32x2", d);
  run<2, 8, 512>("R2 NT8 f32x2", d);
  run<2, 8, 768>("R2 NT8 f32x2", d);
  run<4, 8, 256>("R4 NT8 f32x2", d);
  run<4, 8, 512>("R4 NT8 f32x2", d);
  run<4, 4, 512>("R4 NT4 f32x2", d);
  run<2, 10, 768>("R2 NT10 f32x2", d);
  return 0;
}
