// lds_cost_probe.cu -- how many cycles of an SM's shared-memory pipe one warp-wide LDS.32 / LDS.64 /
// LDS.128 costs for a given lane -> address pattern (B200, sm_100a).  The K3 lane mapping
// (k3_mlp_fp32.cuh) was chosen from this table; output of one run: profiles/r1c_probes.md.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o lds_cost_probe lds_cost_probe.cu && ./lds_cost_probe
//
// 148 CTAs x 16 warps issue 16 * ITERS volatile loads each; SM cycles per warp instruction =
// elapsed (CUDA events) * 1.965 GHz / (16 * ITERS * 16 warps).
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

template <int W>   // words per lane: 1, 2, 4
__global__ void probe(const int* __restrict__ offs, float* out, int iters) {
  extern __shared__ __align__(16) float sm[];
  for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = (float)i;
  __syncthreads();
  const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm) + offs[threadIdx.x & 31];
  float a0 = 0, a1 = 0, a2 = 0, a3 = 0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const uint32_t ad = base + u * 1024;
      if (W == 4) {
        float4 v;
        asm volatile("ld.volatile.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(ad));
        a0 += v.x; a1 += v.y; a2 += v.z; a3 += v.w;
      } else if (W == 2) {
        float2 v;
        asm volatile("ld.volatile.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(ad));
        a0 += v.x; a1 += v.y;
      } else {
        float v;
        asm volatile("ld.volatile.shared.f32 %0, [%1];" : "=f"(v) : "r"(ad));
        a0 += v;
      }
    }
  }
  if (a0 + a1 + a2 + a3 == 12345.f) out[0] = 1.f;
}

struct Pattern { const char* name; int (*byte_offset)(int lane); int align; };

int main() {
  int* d_off; float* d_out;
  cudaMalloc(&d_off, 128); cudaMalloc(&d_out, 16);
  const Pattern pats[] = {
      {"all lanes one address", [](int) { return 0; }, 16},
      {"16*(l/2)   16 addresses, equal lanes adjacent", [](int l) { return 16 * (l / 2); }, 16},
      {"16*(l/4)    8 addresses, equal lanes adjacent", [](int l) { return 16 * (l / 4); }, 16},
      {"656*(l/4)   8 rows of 164 floats, adjacent", [](int l) { return 656 * (l / 4); }, 16},
      {"16*(l/8)    4 addresses, equal lanes adjacent", [](int l) { return 16 * (l / 8); }, 16},
      {"16*(l/16)   2 addresses, equal lanes adjacent", [](int l) { return 16 * (l / 16); }, 16},
      {"16*(l%2)    2 addresses, alternating", [](int l) { return 16 * (l % 2); }, 16},
      {"16*(l%4)    4 addresses, cyclic", [](int l) { return 16 * (l % 4); }, 16},
      {"16*(l%8)    8 addresses, cyclic", [](int l) { return 16 * (l % 8); }, 16},
      {"656*(l%8)   8 rows of 164 floats, cyclic", [](int l) { return 656 * (l % 8); }, 16},
      {"16*l       32 addresses (512 B)", [](int l) { return 16 * l; }, 16},
      {"8*l        32 addresses (256 B)", [](int l) { return 8 * l; }, 8},
      {"8*(l/4)     8 addresses, adjacent", [](int l) { return 8 * (l / 4); }, 8},
      {"8*(l%4)     4 addresses, cyclic", [](int l) { return 8 * (l % 4); }, 8},
      {"4*l        32 addresses (128 B)", [](int l) { return 4 * l; }, 4},
  };
  cudaFuncSetAttribute(probe<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  cudaFuncSetAttribute(probe<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  cudaFuncSetAttribute(probe<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  const int iters = 2048, warps = 16;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  printf("%-50s %8s %8s %8s   (SM cycles per warp instruction at 1.965 GHz)\n", "lane -> byte offset", "LDS.32", "LDS.64", "LDS.128");
  for (const Pattern& p : pats) {
    int h[32];
    for (int l = 0; l < 32; ++l) h[l] = p.byte_offset(l);
    cudaMemcpy(d_off, h, 128, cudaMemcpyHostToDevice);
    printf("%-50s", p.name);
    for (int w = 1; w <= 4; w *= 2) {
      if (p.align < 4 * w) { printf(" %8s", "-"); continue; }
      float ms = 0;
      for (int rep = 0; rep < 2; ++rep) {
        cudaEventRecord(e0);
        if (w == 1) probe<1><<<148, warps * 32, 65536>>>(d_off, d_out, iters);
        if (w == 2) probe<2><<<148, warps * 32, 65536>>>(d_off, d_out, iters);
        if (w == 4) probe<4><<<148, warps * 32, 65536>>>(d_off, d_out, iters);
        cudaEventRecord(e1);
        cudaDeviceSynchronize();
        cudaEventElapsedTime(&ms, e0, e1);
      }
      printf(" %8.2f", ms * 1e-3 * 1.965e9 / (iters * 16.0 * warps));
    }
    printf("\n");
  }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
  return 0;
}
