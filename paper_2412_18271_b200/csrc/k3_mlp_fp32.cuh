// k3_mlp_fp32.cuh -- K3 (FP32 FFMA path: batches below the tensor-core threshold, and on request): per-element MLP 384->160->128->96->1
// with CELU(0.1), forward and input-gradient backward, fused per row tile
// (O5; backward = PAPER.md:67 "forces by backprop", weight gradients
// are never needed).
//
// Rows are atoms of ONE element (element blocks are padded to ROW_PAD = 128 rows), so a
// tile is a dense [128 x K] x [K x N] contraction chain -- a grouped GEMM over the four
// element blocks.  Tile height TM is a template parameter (16, 32, 64, 128; pfc_create picks it,
// measurements in pfc_api.cu); 8 warps per (up to) 64 rows.
// A warp owns min(TM,64) rows x N/8 columns: lane = (row group rg = lane/2, column group
// cg = lane%2), thread rows 64*half + rg + 16r (r < R = min(TM,64)/16), thread columns: float4s at
// 4*cgi + 64*f (f < N/64) plus, for N = 160 / 96, two more at 64*(N/64) + 2*cgi, cgi = 2*(warp%8) + cg.
// The lane mapping is chosen for the shared-memory pipe, which is what bounds this kernel (ncu:
// 84 % of the LSU wavefront peak with the earlier rg = lane/4, cg = lane%4 mapping).  Measured on
// B200 (profiles/r1c_probes.md): an LDS.128 costs 2 cycles of the SM's shared-memory
// pipe when lanes with equal addresses are adjacent (or there are only two addresses, alternating),
// 4 cycles otherwise; with 16 row groups of two adjacent lanes BOTH operand loads are 2-cycle.
//   * the 32-row kernel (the one large batches run) issues the FMAs as packed fma.rn.f32x2
//     (SASS FFMA2): an accumulator PAIR per output holds the sums over even and over odd k, the
//     activation pair comes straight from the float4 along k, the weight pair from the layout
//     B[k/2][n][k%2] pfc_create writes; the pair is added once per phase.  Half the FMA issue slots,
//     which pays at two CTAs per SM (116 registers) with 32-wide K chunks: 2.11 -> 1.96 ms;
//   * activations h1/h2/h3 (later delta1/2/3) stay in shared memory, row-major with row stride
//     = 4 mod 32 floats, so the eight row groups of a half warp read eight different bank groups;
//   * the AEV tile is NOT held: phase 0 streams it in K chunks with cp.async (into the h2/h3
//     region, idle at that time) next to the weight chunks;
//   * a weight chunk (KC k of one phase, all N columns) is one contiguous block fetched from L2 by
//     ONE cp.async.bulk (TMA) on an mbarrier, double buffered, one CTA barrier per chunk; for
//     batches of few tiles per SM an 8-stage full/empty mbarrier ring without CTA barriers inside a
//     phase (DEEP) -- with several CTAs per SM the ring is slower (2.30 vs 2.18 ms at 128 rows);
//   * warps whose 64 rows are all padding skip the arithmetic.
#pragma once
#include "pfc_common.cuh"
#include "tc_ptx.cuh"

namespace pfc {

constexpr int MLP_LD1 = D1 + 4, MLP_LD2 = D2 + 4, MLP_LD3 = D3 + 4;   // row strides (floats): 4 mod 32
// DEEP = false: two staging buffers, one CTA barrier per chunk -- best when several CTAs share an
// SM and hide each other's chunk latency (configs 3 and 4).  DEEP = true: an 8-stage ring guarded
// by full / empty mbarriers with six chunks (60 KB) in flight and no CTA barrier inside a phase --
// for batches of a few tiles per SM, where a tile's time is otherwise 86 chunks x the L2 latency.
template <int TM, bool DEEP = false> struct MlpCfg {                  // TM = 16, 32, 64 or 128 rows per tile
  static constexpr int THREADS = TM >= 64 ? 4 * TM : 256;             // 8 warps per (up to) 64 rows
  static constexpr int WARPS = THREADS / 32;
  static constexpr int R = (TM >= 64 || (TM == 32 && !DEEP)) ? 4 : TM / 16;   // rows per thread
  template <int N> __host__ __device__ static constexpr int nt() { return (TM == 32 && !DEEP) ? N / 32 : N / 16; }   // columns per thread
  static constexpr bool PACKED = TM == 32 && !DEEP;                   // fma.rn.f32x2 inner loop (two CTAs per SM)
  static constexpr int KC = PACKED ? 32 : TM == 64 ? 8 : 16;          // k per staged chunk (64: two CTAs per SM)
  static constexpr int S = DEEP ? 8 : 2;                              // staging buffers
  static constexpr int LEAD = DEEP ? 6 : 1;                           // chunks issued ahead of the consumers
  static constexpr int AS_LD = KC + 4;                                // AEV chunk row stride: 4 mod 8 floats
  static constexpr int AS_FLOATS = TM * AS_LD;                        // one AEV chunk [TM][KC+4]
  static constexpr int BS_FLOATS = KC * D1;                           // one weight buffer (widest N = 160)
  static constexpr size_t SMEM = sizeof(float) * ((size_t)TM * (MLP_LD1 + MLP_LD2 + MLP_LD3) +
                                                  S * BS_FLOATS + (size_t)TM * 8) + 3 * S * 8 + 64;
  static_assert(S * AS_FLOATS <= TM * (MLP_LD2 + MLP_LD3), "AEV chunks live in the h2 + h3 regions during phase 0");
  static_assert((D0 / KC) % S == 0, "phase 0 ends on a ring boundary (full / fullA parity bookkeeping)");
  static_assert(!DEEP || TM <= 32, "the deep ring is for small tiles");
};

// weight image per element (floats): phases 0..5, each B[K][N] row-major
constexpr int MLP_P_OFF0 = 0;                          // W1^T  K=384 N=160
constexpr int MLP_P_OFF1 = MLP_P_OFF0 + D0 * D1;       // W2^T  K=160 N=128
constexpr int MLP_P_OFF2 = MLP_P_OFF1 + D1 * D2;       // W3^T  K=128 N=96
constexpr int MLP_P_OFF3 = MLP_P_OFF2 + D2 * D3;       // W3    K=96  N=128
constexpr int MLP_P_OFF4 = MLP_P_OFF3 + D3 * D2;       // W2    K=128 N=160
constexpr int MLP_P_OFF5 = MLP_P_OFF4 + D2 * D1;       // W1    K=160 N=3x128 (pass-major)
constexpr int MLP_P_FLOATS = MLP_P_OFF5 + D1 * D0;     // 188,416
constexpr int MLP_V_B1 = 0, MLP_V_B2 = D1, MLP_V_B3 = D1 + D2, MLP_V_W4 = D1 + D2 + D3,
              MLP_V_B4 = D1 + D2 + 2 * D3, MLP_V_FLOATS = 484;

// d += a * b on two fp32 lanes (sm_100: SASS FFMA2)
__device__ __forceinline__ void ffma2(float2& d, float2 a, float2 b) {
  unsigned long long ua = *reinterpret_cast<unsigned long long*>(&a), ub = *reinterpret_cast<unsigned long long*>(&b),
                     ud = *reinterpret_cast<unsigned long long*>(&d);
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(ud) : "l"(ua), "l"(ub));
  d = *reinterpret_cast<float2*>(&ud);
}

struct MlpParams {
  const float* wpack[NSPEC];   // MLP_P_FLOATS per element
  const float* vec[NSPEC];     // b1 b2 b3 w4 b4
  int row_start[NSPEC + 1];    // element block boundaries in padded row order
  int row_end[NSPEC];          // row_start[e] + number of atoms of element e
};

__device__ __forceinline__ float celu_f(float x) {
  return x > 0.0f ? x : CELU_ALPHA * (expf(x * (1.0f / CELU_ALPHA)) - 1.0f);
}
// CELU'(z) recovered from h = CELU(z): 1 for h > 0, exp(z/alpha) = h/alpha + 1 otherwise
__device__ __forceinline__ float dcelu_from_h(float h) {
  return h > 0.0f ? 1.0f : fmaf(h, 1.0f / CELU_ALPHA, 1.0f);
}

__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint64_t* bar) {   // arrives when my cp.asyncs landed
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(tc::smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(tc::smem_u32(bar)), "r"(bytes)
               : "memory");
}

// Shared-memory staging state, uniform across the CTA.  Chunk g (counted over the whole tile)
// uses buffer g % S.  full[st] (count 1: the TMA issuer) completes when the weight chunk has landed.
// Deep ring only: fullA[st] (count THREADS: every thread's cp.async granules of the AEV chunk,
// phase 0) and empty[st] (count WARPS: every warp has finished reading the buffer); a chunk is
// issued LEAD = S - 2 chunks ahead, into the buffer released two chunks ago, so warps may drift
// one chunk apart without stalling.
struct MlpPipe {
  float* Bs;                   // [S][BS_FLOATS]
  float* As;                   // [S][AS_FLOATS]  (phase 0 only)
  uint64_t *full, *fullA, *empty;
  uint32_t gc;                 // chunks consumed so far
};

// column c (< N/16) of the thread with column slot cgi (< 16)
template <int N>
__device__ __forceinline__ int mlp_col(int cgi, int c) {
  constexpr int NF4 = N / 64;
  return c < 4 * NF4 ? 64 * (c >> 2) + 4 * cgi + (c & 3) : 64 * NF4 + 2 * cgi + (c - 4 * NF4);
}

// Which rows and columns a thread owns.
//   default: 8 column warps per (up to) 64 rows; lane = (row group lane/2, column slot lane%2);
//            rows 64*(w/8) + lane/2 + 16r, columns mlp_col<N>(2*(w%8) + lane%2, c).
//   PACKED (32 rows): 4 row warps x 2 column warps; lane = (column slot lane/2, row group lane%2);
//            rows 8*(w/2) + 4*(lane%2) + r (r < 4); column slot ct = 16*(w%2) + lane/2 (< 32) owns the
//            pairs {2ct, 2ct+1} + 64f (f < (N/32)/2) and, for N = 160 / 96, the single 64*((N/32)/2) + ct.
//            Per 4 k a warp then spends 2*4 shared-memory pipe cycles on the activations and
//            2*(2,2,1) + (1,0,1) per k pair on the weights: 18 / 16 / 14 for N = 160 / 128 / 96, against
//            24 / 20 / 16 with the default mapping at two rows per thread -- the kernel is bound by
//            that pipe once the FMAs are packed (ncu: 77 % of its peak).
template <int TM, bool DEEP> struct MlpLane {
  static constexpr bool PACKED = MlpCfg<TM, DEEP>::PACKED;
  int lane, w;
  __device__ __forceinline__ MlpLane() : lane(threadIdx.x & 31), w(threadIdx.x >> 5) {}
  __device__ __forceinline__ int ct() const { return PACKED ? 16 * (w & 1) + (lane >> 1) : 2 * (w & 7) + (lane & 1); }
  __device__ __forceinline__ int row(int r) const {
    return PACKED ? 8 * (w >> 1) + 4 * (lane & 1) + r : 64 * (w >> 3) + (lane >> 1) + 16 * r;
  }
  __device__ __forceinline__ int warp_row0() const { return PACKED ? 8 * (w >> 1) : 64 * (w >> 3); }
  template <int N> __device__ __forceinline__ int col(int c) const {
    if (PACKED) {
      constexpr int NW = (N / 32) / 2;
      return c < 2 * NW ? 64 * (c >> 1) + 2 * ct() + (c & 1) : 64 * NW + ct();
    }
    return mlp_col<N>(ct(), c);
  }
};

// acc[r][c] = sum_k A[rowbase + 16r][k] * B[k][mlp_col<N>(cgi, c)],  k < K, r < R,  rowbase = 64*half + rg.
// A_GLOBAL: A is the AEV tile in global memory (row stride AEV_LEN), streamed; else A is a
// row-major shared-memory activation with row stride lda.
template <int TM, bool DEEP, int K, int N, bool A_GLOBAL>
__device__ __forceinline__ void mlp_gemm(MlpPipe& P, const float* __restrict__ A, int lda,
                                         const float* __restrict__ Bg, bool active,
                                         float (&acc)[MlpCfg<TM, DEEP>::R][MlpCfg<TM, DEEP>::template nt<N>()]) {
  using Cfg = MlpCfg<TM, DEEP>;
  constexpr int NT = Cfg::template nt<N>();
  constexpr int NF4 = N / 64;                            // float4 column groups per thread
  constexpr bool HAS2 = (N % 64) == 32;                  // plus one float2 group (N = 160, 96)
  constexpr int R = Cfg::R, S = Cfg::S, LEAD = Cfg::LEAD;
  constexpr int MLP_KC = Cfg::KC, MLP_AS_LD = Cfg::AS_LD, MLP_BS_FLOATS = Cfg::BS_FLOATS;
  constexpr int NCH = K / MLP_KC;
  constexpr int GR = MLP_KC / 4;                         // 16-byte granules per AEV chunk row
  constexpr uint32_t CH_BYTES = MLP_KC * N * sizeof(float);
  constexpr int AS_FLOATS = Cfg::AS_FLOATS;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int rowbase = 64 * (w >> 3) + (lane >> 1), cgi = 2 * (w & 7) + (lane & 1);
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < NT; ++c) acc[r][c] = 0.0f;
  // the deep ring signals an AEV chunk through fullA (every thread's granules), a weight-only chunk
  // through full; the two-buffer pipeline uses full + cp.async.wait_group + the CTA barrier
  uint64_t* fullb = (DEEP && A_GLOBAL) ? P.fullA : P.full;
  constexpr uint32_t BASE = (DEEP && !A_GLOBAL) ? D0 / MLP_KC : 0;   // chunks before this barrier set's first use
  auto issue = [&](int ch, uint32_t gch) {               // chunk ch of this phase = chunk gch of the tile
    const uint32_t st = gch % S;
    if (tid == 0) {
      if (DEEP && A_GLOBAL) mbar_expect_tx(&fullb[st], CH_BYTES);
      else tc::mbar_arrive_expect_tx(&fullb[st], CH_BYTES);
      tc::bulk_g2s(P.Bs + st * MLP_BS_FLOATS, Bg + (size_t)ch * MLP_KC * N, CH_BYTES, &fullb[st]);
    }
    if (A_GLOBAL) {                                      // TM rows x GR granules
      for (int t = tid; t < GR * TM; t += Cfg::THREADS)
        cp_async16(P.As + st * AS_FLOATS + (t / GR) * MLP_AS_LD + 4 * (t % GR),
                   A + (size_t)(t / GR) * AEV_LEN + ch * MLP_KC + 4 * (t % GR));
      if (DEEP) cp_async_mbar_arrive_noinc(&fullb[st]);
      else cp_async_commit();
    }
  };
  // PACKED (the 32-row kernel): accumulator pairs (sum over even k, sum over odd k) advanced by one
  // fma.rn.f32x2 (SASS FFMA2) per pair -- half the FMA issue slots; the pair is added at the end.
  // Otherwise one accumulator, k ascending.
  constexpr bool PACKED = Cfg::PACKED;
  float2 acc2[PACKED ? R : 1][PACKED ? NT : 1];
  if (PACKED) {
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
      for (int c = 0; c < NT; ++c) acc2[PACKED ? r : 0][PACKED ? c : 0] = make_float2(0.0f, 0.0f);
  }
  auto compute = [&](int ch, uint32_t st) {
    const float* bs = P.Bs + st * MLP_BS_FLOATS;
    if constexpr (PACKED) {                              // MlpLane's PACKED mapping
      constexpr int NW = NT / 2;
      constexpr bool SINGLE = (NT & 1) != 0;
      const int ct = 16 * (w & 1) + (lane >> 1), r0 = 8 * (w >> 1) + 4 * (lane & 1);
      const float* at = A_GLOBAL ? P.As + st * AS_FLOATS + r0 * MLP_AS_LD : A + (size_t)r0 * lda + ch * MLP_KC;
      const int astr = A_GLOBAL ? MLP_AS_LD : lda;
#pragma unroll
      for (int k4 = 0; k4 < MLP_KC / 4; ++k4) {
        float4 a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = *reinterpret_cast<const float4*>(at + r * astr + 4 * k4);
#pragma unroll
        for (int j = 0; j < 2; ++j) {                    // k pair 2*k4 + j of the chunk: B2[pair][n][2]
          const float* brow = bs + (2 * k4 + j) * (2 * N);
          float2 b[NT];
#pragma unroll
          for (int f = 0; f < NW; ++f) {
            const float4 v = *reinterpret_cast<const float4*>(brow + 2 * (64 * f + 2 * ct));
            b[2 * f] = make_float2(v.x, v.y); b[2 * f + 1] = make_float2(v.z, v.w);
          }
          if (SINGLE) b[NT - 1] = *reinterpret_cast<const float2*>(brow + 2 * (64 * NW + ct));
#pragma unroll
          for (int r = 0; r < R; ++r) {
            const float2 av = j == 0 ? make_float2(a[r].x, a[r].y) : make_float2(a[r].z, a[r].w);
#pragma unroll
            for (int c = 0; c < NT; ++c) ffma2(acc2[PACKED ? r : 0][PACKED ? c : 0], av, b[c]);
          }
        }
      }
    } else {
    const float* at = A_GLOBAL ? P.As + st * AS_FLOATS + rowbase * MLP_AS_LD
                               : A + (size_t)rowbase * lda + ch * MLP_KC;
    const int astr = 16 * (A_GLOBAL ? MLP_AS_LD : lda);
#pragma unroll
    for (int k4 = 0; k4 < MLP_KC / 4; ++k4) {
      float4 a[R];
#pragma unroll
      for (int r = 0; r < R; ++r) a[r] = *reinterpret_cast<const float4*>(at + r * astr + 4 * k4);
#pragma unroll
      for (int j = 0; j < 2; ++j) {                      // k pair 2*k4 + j of the chunk: B2[pair][n][2]
        const float* brow = bs + (2 * k4 + j) * (2 * N);
        float2 b[NT];
#pragma unroll
        for (int f = 0; f < NF4; ++f) {
          const float4 v0 = *reinterpret_cast<const float4*>(brow + 2 * (64 * f + 4 * cgi));
          const float4 v1 = *reinterpret_cast<const float4*>(brow + 2 * (64 * f + 4 * cgi) + 4);
          b[4 * f] = make_float2(v0.x, v0.y); b[4 * f + 1] = make_float2(v0.z, v0.w);
          b[4 * f + 2] = make_float2(v1.x, v1.y); b[4 * f + 3] = make_float2(v1.z, v1.w);
        }
        if (HAS2) {
          const float4 v = *reinterpret_cast<const float4*>(brow + 2 * (64 * NF4 + 2 * cgi));
          b[NT - 2] = make_float2(v.x, v.y); b[NT - 1] = make_float2(v.z, v.w);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const float2 av = j == 0 ? make_float2(a[r].x, a[r].y) : make_float2(a[r].z, a[r].w);
#pragma unroll
          for (int c = 0; c < NT; ++c) {
            if (PACKED) {
              ffma2(acc2[PACKED ? r : 0][PACKED ? c : 0], av, b[c]);
            } else {
              acc[r][c] = fmaf(av.x, b[c].x, acc[r][c]);
              acc[r][c] = fmaf(av.y, b[c].y, acc[r][c]);
            }
          }
        }
      }
    }
    }
  };
  __syncthreads();                  // previous phase: activation stores visible, every staging buffer released
  if constexpr (!DEEP) {
    issue(0, P.gc);
    for (int ch = 0; ch < NCH; ++ch) {
      const uint32_t st = P.gc & 1u;
      if (A_GLOBAL) cp_async_wait<0>();
      tc::mbar_wait(&P.full[st], (P.gc >> 1) & 1u);
      __syncthreads();              // all A granules visible; the other buffer is no longer read
      if (ch + 1 < NCH) issue(ch + 1, P.gc + 1);
      ++P.gc;
      if (active) compute(ch, st);
    }
  } else {
#pragma unroll
    for (int c = 0; c < LEAD && c < NCH; ++c) issue(c, P.gc + c);
#pragma unroll 1
    for (int ch = 0; ch < NCH; ++ch) {
      const uint32_t gch = P.gc, st = gch % S;
      if (ch + LEAD < NCH) {
        if (ch >= S - LEAD) {       // the target buffer was last read as chunk gch + LEAD - S of this phase
          const uint32_t gp = gch + LEAD - S;
          tc::mbar_wait(&P.empty[gp % S], (gp / S) & 1u);
        }
        issue(ch + LEAD, gch + LEAD);
      }
      tc::mbar_wait(&fullb[st], ((gch - BASE) / S) & 1u);
      ++P.gc;
      if (active) compute(ch, st);
      __syncwarp();                 // every lane's reads of this buffer are done
      if (lane == 0) tc::mbar_arrive(&P.empty[st]);
    }
  }
  if (PACKED) {
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
      for (int c = 0; c < NT; ++c) acc[r][c] = acc2[PACKED ? r : 0][PACKED ? c : 0].x + acc2[PACKED ? r : 0][PACKED ? c : 0].y;
  }
}

template <int TM, bool DEEP>
__global__ void __launch_bounds__(MlpCfg<TM, DEEP>::THREADS, (TM == 64 || MlpCfg<TM, DEEP>::PACKED) ? 2 : 1)
k3_mlp_fp32_kernel(const __grid_constant__ MlpParams P, const float* __restrict__ aev,
                   float* __restrict__ g, float* __restrict__ e_row) {
  extern __shared__ __align__(16) float smem[];
  float* H1 = smem;                                   // [TM][LD1]  h1, later delta1
  float* H2 = H1 + TM * MLP_LD1;                      // [TM][LD2]  h2, later delta2 (phase 0: AEV chunks, into h3)
  float* H3 = H2 + TM * MLP_LD2;                      // [TM][LD3]  delta3
  using Cfg = MlpCfg<TM, DEEP>;
  MlpPipe pipe;
  pipe.Bs = H3 + TM * MLP_LD3;
  pipe.As = H2;
  float* esum = pipe.Bs + Cfg::S * Cfg::BS_FLOATS;    // [TM][8] partial energies per column group
  pipe.full = reinterpret_cast<uint64_t*>(esum + TM * 8);
  pipe.fullA = pipe.full + Cfg::S;
  pipe.empty = pipe.fullA + Cfg::S;
  pipe.gc = 0;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  constexpr int R = Cfg::R;
  constexpr bool PACKED = Cfg::PACKED;
  const MlpLane<TM, DEEP> L;
  const int row0 = blockIdx.x * TM;
  int el = 0;
#pragma unroll
  for (int k = 1; k < NSPEC; ++k) el += (row0 >= P.row_start[k]);
  const float* __restrict__ Wp = P.wpack[el];
  const float* __restrict__ V = P.vec[el];
  if (row0 >= P.row_end[el]) return;                  // a tile of padding only (CTA-uniform)
  const bool active = row0 + L.warp_row0() < P.row_end[el];   // warp-uniform: my warp's rows hold an atom
  if (tid == 0) {
    for (int st = 0; st < Cfg::S; ++st) {
      tc::mbar_init(&pipe.full[st], 1);
      tc::mbar_init(&pipe.fullA[st], Cfg::THREADS);
      tc::mbar_init(&pipe.empty[st], Cfg::WARPS);
    }
    tc::mbar_fence_init();
  }
  // (the first __syncthreads of mlp_gemm orders the init before any use)

  // ---- forward ----
  {
    constexpr int NT = Cfg::template nt<D1>();
    float acc[R][NT];
    mlp_gemm<TM, DEEP, D0, D1, true>(pipe, aev + (size_t)row0 * AEV_LEN, 0, Wp + MLP_P_OFF0, active, acc);
    if (active) {
#pragma unroll
      for (int c = 0; c < NT; ++c) {
        const int n = L.template col<D1>(c);
        const float bias = __ldg(V + MLP_V_B1 + n);
#pragma unroll
        for (int r = 0; r < R; ++r) H1[L.row(r) * MLP_LD1 + n] = celu_f(acc[r][c] + bias);
      }
    }
  }
  {
    constexpr int NT = Cfg::template nt<D2>();
    float acc[R][NT];
    mlp_gemm<TM, DEEP, D1, D2, false>(pipe, H1, MLP_LD1, Wp + MLP_P_OFF1, active, acc);
    if (active) {
#pragma unroll
      for (int c = 0; c < NT; ++c) {
        const int n = L.template col<D2>(c);
        const float bias = __ldg(V + MLP_V_B2 + n);
#pragma unroll
        for (int r = 0; r < R; ++r) H2[L.row(r) * MLP_LD2 + n] = celu_f(acc[r][c] + bias);
      }
    }
  }
  {
    constexpr int NT = Cfg::template nt<D3>();
    float acc[R][NT];
    mlp_gemm<TM, DEEP, D2, D3, false>(pipe, H2, MLP_LD2, Wp + MLP_P_OFF2, active, acc);
    float part[R];
#pragma unroll
    for (int r = 0; r < R; ++r) part[r] = 0.0f;
    if (active) {
#pragma unroll
      for (int c = 0; c < NT; ++c) {
        const int n = L.template col<D3>(c);
        const float bias = __ldg(V + MLP_V_B3 + n), w4 = __ldg(V + MLP_V_W4 + n);
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const float h = celu_f(acc[r][c] + bias);
          part[r] = fmaf(w4, h, part[r]);
          H3[L.row(r) * MLP_LD3 + n] = w4 * dcelu_from_h(h);   // delta3 = dE/dz3
        }
      }
    }
    // e_i = b4 + sum over the 96 columns: the lanes that share my rows (fixed xor tree), then the
    // column warps in a fixed order
#pragma unroll
    for (int r = 0; r < R; ++r) {
      float s = part[r];
      if (PACKED) {
        s += __shfl_xor_sync(0xffffffffu, s, 2); s += __shfl_xor_sync(0xffffffffu, s, 4);
        s += __shfl_xor_sync(0xffffffffu, s, 8); s += __shfl_xor_sync(0xffffffffu, s, 16);
        if (lane < 2) esum[L.row(r) * 8 + (w & 1)] = s;
      } else {
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        if ((lane & 1) == 0) esum[L.row(r) * 8 + (w & 7)] = s;
      }
    }
    __syncthreads();
    if (tid < TM && row0 + tid < P.row_end[el]) {
      const float* p = esum + tid * 8;
      const float sum = PACKED ? p[0] + p[1] : ((p[0] + p[1]) + (p[2] + p[3])) + ((p[4] + p[5]) + (p[6] + p[7]));
      e_row[row0 + tid] = sum + __ldg(V + MLP_V_B4);
    }
  }
  // ---- backward (input gradient only) ----
  {
    constexpr int NT = Cfg::template nt<D2>();
    float acc[R][NT];
    mlp_gemm<TM, DEEP, D3, D2, false>(pipe, H3, MLP_LD3, Wp + MLP_P_OFF3, active, acc);
    if (active) {
#pragma unroll
      for (int c = 0; c < NT; ++c)
#pragma unroll
        for (int r = 0; r < R; ++r) {
          float* hp = H2 + L.row(r) * MLP_LD2 + L.template col<D2>(c);
          *hp = acc[r][c] * dcelu_from_h(*hp);          // delta2 over h2 (own elements only)
        }
    }
  }
  {
    constexpr int NT = Cfg::template nt<D1>();
    float acc[R][NT];
    mlp_gemm<TM, DEEP, D2, D1, false>(pipe, H2, MLP_LD2, Wp + MLP_P_OFF4, active, acc);
    if (active) {
#pragma unroll
      for (int c = 0; c < NT; ++c)
#pragma unroll
        for (int r = 0; r < R; ++r) {
          float* hp = H1 + L.row(r) * MLP_LD1 + L.template col<D1>(c);
          *hp = acc[r][c] * dcelu_from_h(*hp);          // delta1
        }
    }
  }
#pragma unroll 1
  for (int pass = 0; pass < D0 / 128; ++pass) {
    float acc[R][Cfg::template nt<128>()];
    mlp_gemm<TM, DEEP, D1, 128, false>(pipe, H1, MLP_LD1, Wp + MLP_P_OFF5 + pass * D1 * 128, active, acc);
    if (active) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        float* dst = g + (size_t)(row0 + L.row(r)) * AEV_LEN + pass * 128;
        if constexpr (PACKED) {
          *reinterpret_cast<float2*>(dst + 2 * L.ct()) = make_float2(acc[r][0], acc[r][1]);
          *reinterpret_cast<float2*>(dst + 64 + 2 * L.ct()) = make_float2(acc[r][2], acc[r][3]);
        } else {
          *reinterpret_cast<float4*>(dst + 4 * L.ct()) = make_float4(acc[r][0], acc[r][1], acc[r][2], acc[r][3]);
          *reinterpret_cast<float4*>(dst + 64 + 4 * L.ct()) = make_float4(acc[r][4], acc[r][5], acc[r][6], acc[r][7]);
        }
      }
    }
  }
}

}  // namespace pfc
