// k3_mlp_cluster.cuh -- K3 for a single small molecule (the regime the paper
// measures: one 9-atom molecule, launch- and latency-bound): the per-element MLP
// 384->160->128->96->1, forward and input-gradient backward in FP32 (O5, O7), with every
// 16-row tile spread over a CLUSTER OF 8 CTAs.
//
// Why.  A batch of a few dozen atoms has one tile per element.  One CTA per tile (k3_mlp_fp32.cuh)
// then walks the element's 1.5 MB of weights alone, chunk by chunk, at one SM's L2 bandwidth: 21 us
// of the 37 us the kernel takes on config 0.  Here the 8 CTAs of a cluster split the OUTPUT columns
// of every layer: CTA r of the cluster computes columns [r N/8, (r+1) N/8) of each of the six GEMM
// phases for all 16 rows, so it needs one eighth of every weight matrix -- 94 KB in all, which fits
// its shared memory and is fetched by six bulk copies (TMA, cp.async.bulk + mbarrier) issued
// TOGETHER at kernel start: the whole weight walk costs one L2 latency.  After each phase the CTAs
// exchange their column slices of the activations through distributed shared memory (each thread
// stores its 4-row x 1-column result into the activation buffer of all 8 CTAs,
// st.shared::cluster) and meet at a cluster barrier.
//
//   phase  input (K)          weights (slice)       output (columns per CTA)
//   0      aev      (384)     W1   [k][20]          h1 = CELU(z1 + b1)                 (160: 20)
//   1      h1       (160)     W2   [k][16]          h2 = CELU(z2 + b2)                 (128: 16)
//   2      h2       (128)     W3   [k][12]          e += w4.CELU(z3 + b3); delta3      ( 96: 12)
//   3      delta3   ( 96)     W3^T [k][16]          delta2 = (.) * CELU'(z2 + b2)      (128: 16)
//   4      delta2   (128)     W2^T [k][20]          delta1 = (.) * CELU'(z1 + b1)      (160: 20)
//   5      delta1   (160)     W1^T [k][48]          g -> global                        (384: 48)
// Activations live TRANSPOSED in shared memory ([k][16 rows]): a thread owns 4 rows x 1 column and,
// per k, reads one weight (consecutive lanes: consecutive columns) and one float4 of activations
// (a broadcast).  K is split over KS thread groups (512 threads: 12 to 80 k per thread) whose partial sums
// are added in a fixed order;
// CELU' of the own columns stays in registers between the forward and the backward phase (the
// thread mapping of phases 0/4 and 1/3 is the same).  The energy is reduced over the 12 columns of
// a CTA and then over the 8 CTAs (into CTA 0's shared memory), both in a fixed order: no atomics,
// bit-reproducible.
#pragma once
#include "k3_mlp_fp32.cuh"

namespace pfc {

constexpr int CL_SIZE = 8;                       // CTAs per cluster (the portable maximum)
constexpr int CL_TM = 16;                        // rows per tile
constexpr int CL_THREADS = 512;
constexpr int CL_MAX_TILES = 18;                 // 18 clusters x 8 CTAs <= 148 SMs: one wave
constexpr int CL_NC0 = D1 / CL_SIZE, CL_NC1 = D2 / CL_SIZE, CL_NC2 = D3 / CL_SIZE, CL_NC3 = D2 / CL_SIZE,
              CL_NC4 = D1 / CL_SIZE, CL_NC5 = D0 / CL_SIZE;     // 20 16 12 16 20 48
constexpr int CL_W0 = 0, CL_W1 = CL_W0 + D0 * CL_NC0, CL_W2 = CL_W1 + D1 * CL_NC1, CL_W3 = CL_W2 + D2 * CL_NC2,
              CL_W4 = CL_W3 + D3 * CL_NC3, CL_W5 = CL_W4 + D2 * CL_NC4, CL_W_FLOATS = CL_W5 + D1 * CL_NC5;   // 23,552
static_assert(CL_W_FLOATS == 23552 && CL_W_FLOATS * CL_SIZE == MLP_P_FLOATS, "weight slices of one CTA");
constexpr int CL_PART = 2048;                    // partial sums: (KS - 1) x (NC x 4 row groups) x 4 rows (largest: 7 x 64 x 4)
constexpr int CL_SCRATCH = CL_PART + CL_TM * CL_NC5;   // + phase 5: the g block [16][48]

struct ClSmem {
  float w[CL_W_FLOATS];                          // my column slices of the six weight matrices, [k][nc] each
  float aevT[D0 * CL_TM];                        // [k][16]
  float h1T[D1 * CL_TM];                         // h1, later delta1
  float h2T[D2 * CL_TM];                         // h2, later delta2
  float d3T[D3 * CL_TM];                         // delta3
  float scratch[CL_SCRATCH];                     // K-split partial sums; phase 5: the g block [16][48]
  float esum[CL_SIZE][CL_TM];                    // CTA 0: energy partials of the 8 CTAs
  float ecol[CL_NC2 * 4][4];                     // energy partials of my 12 columns x 4 row groups
  uint64_t wbar[6];
};
constexpr size_t CL_SMEM_BYTES = sizeof(ClSmem) + 16;

struct ClParams {
  const float* wcl;            // [NSPEC][CL_SIZE][CL_W_FLOATS]
  const float* vec[NSPEC];     // b1 b2 b3 w4 b4 (MLP_V_*)
  int n_tiles;
  int row0[CL_MAX_TILES];      // first padded row of the tile
  int elem[CL_MAX_TILES];
  int rows[CL_MAX_TILES];      // real rows in the tile (1..16)
};

namespace cl {
__device__ __forceinline__ uint32_t cta_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of my shared-memory location `p` in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to(const void* p, uint32_t rank) {
  uint32_t a = tc::smem_u32(p), out;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(out) : "r"(a), "r"(rank));
  return out;
}
__device__ __forceinline__ void st_cluster4(uint32_t addr, float4 v) {
  asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
               : "memory");
}
// my 4 rows of column `col` into the transposed activation buffer `buf` of every CTA of the cluster
__device__ __forceinline__ void broadcast4(float* buf, int col, int rg, float4 v) {
  float* p = buf + col * CL_TM + 4 * rg;
#pragma unroll
  for (uint32_t r = 0; r < CL_SIZE; ++r) st_cluster4(map_to(p, r), v);
}
}  // namespace cl

// acc[0..3] = sum_k actT[k][4 rg + 0..3] * Ws[k][c] over this thread's K split; then the splits are added in
// order.  Returns true for the threads that hold a complete sum (split 0 of an active (c, rg)).
template <int K, int NC, int KS>
__device__ __forceinline__ bool cl_gemm(const float* __restrict__ actT, const float* __restrict__ Ws, float* scratch,
                                        int& c, int& rg, float4& acc) {
  constexpr int PAIRS = NC * 4, KL = K / KS;
  static_assert(K % KS == 0 && KL % 4 == 0 && PAIRS * KS <= CL_THREADS && PAIRS * (KS - 1) * 4 <= CL_PART, "thread / scratch budget");
  const int tid = threadIdx.x, ks = tid / PAIRS, rem = tid - ks * PAIRS;
  c = rem % NC; rg = rem / NC;
  const bool active = ks < KS;
  acc = make_float4(0.f, 0.f, 0.f, 0.f);
  if (active) {
    const float* a = actT + (size_t)ks * KL * CL_TM + 4 * rg;
    const float* w = Ws + (size_t)ks * KL * NC + c;
#pragma unroll 4
    for (int k = 0; k < KL; ++k) {
      const float4 x = *reinterpret_cast<const float4*>(a + k * CL_TM);
      const float wk = w[k * NC];
      acc.x = fmaf(x.x, wk, acc.x); acc.y = fmaf(x.y, wk, acc.y); acc.z = fmaf(x.z, wk, acc.z); acc.w = fmaf(x.w, wk, acc.w);
    }
  }
  if (KS > 1) {
    if (active && ks > 0) *reinterpret_cast<float4*>(scratch + ((ks - 1) * PAIRS + rem) * 4) = acc;
    __syncthreads();
    if (active && ks == 0) {
#pragma unroll
      for (int s = 1; s < KS; ++s) {
        const float4 p = *reinterpret_cast<const float4*>(scratch + ((s - 1) * PAIRS + rem) * 4);
        acc.x += p.x; acc.y += p.y; acc.z += p.z; acc.w += p.w;
      }
    }
  }
  return active && ks == 0;
}

// CELU and CELU', alpha = 0.1, branch-free: e = exp(min(x, 0) / alpha) is exactly 1 for x >= 0
__device__ __forceinline__ float cl_dcelu(float x) { return ex2_approx(fminf(x, 0.0f) * (LOG2E / CELU_ALPHA)); }
__device__ __forceinline__ float cl_celu(float x) { return fmaxf(x, 0.0f) + fmaf(CELU_ALPHA, cl_dcelu(x), -CELU_ALPHA); }

__global__ void __cluster_dims__(CL_SIZE, 1, 1) __launch_bounds__(CL_THREADS, 1)
k3_mlp_cluster_kernel(const __grid_constant__ ClParams P, const float* __restrict__ aev, float* __restrict__ g,
                      float* __restrict__ e_row) {
  extern __shared__ __align__(16) uint8_t cl_smem_raw[];
  ClSmem& S = *reinterpret_cast<ClSmem*>(cl_smem_raw);      // (no integer round trip: the accesses stay LDS / STS)
  const int tid = threadIdx.x;
  const uint32_t rank = cl::cta_rank();
  const int tile = blockIdx.x / CL_SIZE;
  const int el = P.elem[tile], row0 = P.row0[tile], n_real = P.rows[tile];
  const float* V = P.vec[el];

  // ---- all six weight slices in flight at once ----
  if (tid == 0) {
    for (int p = 0; p < 6; ++p) tc::mbar_init(&S.wbar[p], 1);
    tc::mbar_fence_init();
    const float* src = P.wcl + ((size_t)el * CL_SIZE + rank) * CL_W_FLOATS;
    const int off[7] = {CL_W0, CL_W1, CL_W2, CL_W3, CL_W4, CL_W5, CL_W_FLOATS};
    for (int p = 0; p < 6; ++p) {
      const uint32_t bytes = (uint32_t)(off[p + 1] - off[p]) * sizeof(float);
      tc::mbar_arrive_expect_tx(&S.wbar[p], bytes);
      tc::bulk_g2s(S.w + off[p], src + off[p], bytes, &S.wbar[p]);
    }
  }
  // ---- the tile's AEV rows, transposed (rows beyond n_real are zero: K2 never writes padded rows) ----
  for (int q = tid; q < CL_TM * (D0 / 4); q += CL_THREADS) {
    const int r = q / (D0 / 4), k4 = q - r * (D0 / 4);
    const float4 v = r < n_real ? __ldg(reinterpret_cast<const float4*>(aev + (size_t)(row0 + r) * AEV_LEN) + k4)
                                : make_float4(0.f, 0.f, 0.f, 0.f);
    S.aevT[(4 * k4 + 0) * CL_TM + r] = v.x; S.aevT[(4 * k4 + 1) * CL_TM + r] = v.y;
    S.aevT[(4 * k4 + 2) * CL_TM + r] = v.z; S.aevT[(4 * k4 + 3) * CL_TM + r] = v.w;
  }
  __syncthreads();                               // aevT complete, barriers initialised
  int c, rg;
  float4 acc;
  float4 dc1 = make_float4(0.f, 0.f, 0.f, 0.f), dc2 = dc1;   // CELU' of my columns of z1 / z2

  // ---- phase 0: h1 ----
  tc::mbar_wait(&S.wbar[0], 0);
  const bool own0 = cl_gemm<D0, CL_NC0, 6>(S.aevT, S.w + CL_W0, S.scratch, c, rg, acc);
  cl::cluster_sync();                            // every CTA of the cluster is running: its shared memory may be written
  if (own0) {
    const int n = (int)rank * CL_NC0 + c;
    const float b = __ldg(V + MLP_V_B1 + n);
    const float4 z = make_float4(acc.x + b, acc.y + b, acc.z + b, acc.w + b);
    dc1 = make_float4(cl_dcelu(z.x), cl_dcelu(z.y), cl_dcelu(z.z), cl_dcelu(z.w));
    cl::broadcast4(S.h1T, n, rg, make_float4(cl_celu(z.x), cl_celu(z.y), cl_celu(z.z), cl_celu(z.w)));
  }
  cl::cluster_sync();
  // ---- phase 1: h2 ----
  tc::mbar_wait(&S.wbar[1], 0);
  if (cl_gemm<D1, CL_NC1, 8>(S.h1T, S.w + CL_W1, S.scratch, c, rg, acc)) {
    const int n = (int)rank * CL_NC1 + c;
    const float b = __ldg(V + MLP_V_B2 + n);
    const float4 z = make_float4(acc.x + b, acc.y + b, acc.z + b, acc.w + b);
    dc2 = make_float4(cl_dcelu(z.x), cl_dcelu(z.y), cl_dcelu(z.z), cl_dcelu(z.w));
    cl::broadcast4(S.h2T, n, rg, make_float4(cl_celu(z.x), cl_celu(z.y), cl_celu(z.z), cl_celu(z.w)));
  }
  cl::cluster_sync();
  // ---- phase 2: energy and delta3 ----
  tc::mbar_wait(&S.wbar[2], 0);
  if (cl_gemm<D2, CL_NC2, 8>(S.h2T, S.w + CL_W2, S.scratch, c, rg, acc)) {
    const int n = (int)rank * CL_NC2 + c;
    const float b = __ldg(V + MLP_V_B3 + n), w4 = __ldg(V + MLP_V_W4 + n);
    const float4 z = make_float4(acc.x + b, acc.y + b, acc.z + b, acc.w + b);
    *reinterpret_cast<float4*>(S.ecol[rg * CL_NC2 + c]) =
        make_float4(w4 * cl_celu(z.x), w4 * cl_celu(z.y), w4 * cl_celu(z.z), w4 * cl_celu(z.w));
    cl::broadcast4(S.d3T, n, rg, make_float4(w4 * cl_dcelu(z.x), w4 * cl_dcelu(z.y), w4 * cl_dcelu(z.z), w4 * cl_dcelu(z.w)));
  }
  __syncthreads();
  if (tid < CL_TM) {                             // my 12 columns, in order, into CTA 0's table
    float s = 0.0f;
    for (int cc = 0; cc < CL_NC2; ++cc) s += S.ecol[(tid >> 2) * CL_NC2 + cc][tid & 3];
    const uint32_t dst = cl::map_to(&S.esum[rank][tid], 0);
    asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(dst), "f"(s) : "memory");
  }
  cl::cluster_sync();
  if (rank == 0 && tid < n_real) {               // the 8 CTAs, in order
    float s = 0.0f;
    for (int r = 0; r < CL_SIZE; ++r) s += S.esum[r][tid];
    e_row[row0 + tid] = s + __ldg(V + MLP_V_B4);
  }
  // ---- phase 3: delta2 ----
  tc::mbar_wait(&S.wbar[3], 0);
  if (cl_gemm<D3, CL_NC3, 8>(S.d3T, S.w + CL_W3, S.scratch, c, rg, acc)) {
    const int n = (int)rank * CL_NC3 + c;
    cl::broadcast4(S.h2T, n, rg, make_float4(acc.x * dc2.x, acc.y * dc2.y, acc.z * dc2.z, acc.w * dc2.w));
  }
  cl::cluster_sync();
  // ---- phase 4: delta1 ----
  tc::mbar_wait(&S.wbar[4], 0);
  if (cl_gemm<D2, CL_NC4, 4>(S.h2T, S.w + CL_W4, S.scratch, c, rg, acc)) {
    const int n = (int)rank * CL_NC4 + c;
    cl::broadcast4(S.h1T, n, rg, make_float4(acc.x * dc1.x, acc.y * dc1.y, acc.z * dc1.z, acc.w * dc1.w));
  }
  cl::cluster_sync();
  // ---- phase 5: g, my 48 columns of the 16 rows ----
  tc::mbar_wait(&S.wbar[5], 0);
  if (cl_gemm<D1, CL_NC5, 2>(S.h1T, S.w + CL_W5, S.scratch, c, rg, acc)) {
    float* blk = S.scratch + CL_PART;
    blk[(4 * rg + 0) * CL_NC5 + c] = acc.x; blk[(4 * rg + 1) * CL_NC5 + c] = acc.y;
    blk[(4 * rg + 2) * CL_NC5 + c] = acc.z; blk[(4 * rg + 3) * CL_NC5 + c] = acc.w;
  }
  __syncthreads();
  for (int q = tid; q < n_real * (CL_NC5 / 4); q += CL_THREADS) {
    const int r = q / (CL_NC5 / 4), c4 = q - r * (CL_NC5 / 4);
    *reinterpret_cast<float4*>(g + (size_t)(row0 + r) * AEV_LEN + (int)rank * CL_NC5 + 4 * c4) =
        *reinterpret_cast<const float4*>(S.scratch + CL_PART + r * CL_NC5 + 4 * c4);
  }
}

}  // namespace pfc
