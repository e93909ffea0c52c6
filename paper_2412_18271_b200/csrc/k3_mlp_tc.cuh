// k3_mlp_tc.cuh -- K3 (tensor-core path): the per-element MLP 384->160->128->96->1, forward and
// input-gradient backward, as a chain of eight grouped-GEMM phases per 128-row tile on the
// tcgen05 tensor cores (O5 / section 5; backward = PAPER.md:67 "forces by backprop").
//
// Precision: kind::f16 with a 3-term split and fp32 accumulation in TMEM,
//     A*B ~= A_hi*B_hi + A_lo*B_hi + A_hi*B_lo,   x_hi = fp16(x),  x_lo = fp16(x - x_hi):
// 11 + 11 significant bits per operand (x - x_hi is exact in fp32; the tensor core multiplies
// fp16 subnormals exactly -- measured -- so a small remainder costs absolute, not relative,
// accuracy: 3e-8 of the operand's scale).  Every operand class is pre-scaled by an exact power of
// two that puts its typical magnitude well inside fp16's range (weights per layer and element from
// max|W|, the AEV by 8, the backward deltas from max|w4|); the scales leave through the epilogue
// factor of each phase (ks[q] in the per-element table), so no rounding is added.  Against the round-1 kind::tf32
// split this is half the tensor-pipe time per k (K = 16 per MMA instead of 8), half the operand
// bytes in shared memory and in the weight stream.  (A bf16 remainder would not need the scaling,
// but the hardware rejects instruction descriptors that mix fp16 and bf16 operands -- measured.)
// N_TERMS = 1 is plain FP16 operands, kept only to produce the evidence that a single 16-bit
// term misses the tolerance.
//
// One persistent CTA per SM, 608 threads, 128-row tiles of ONE element each:
//   warps 0-15 workers (warp = TMEM lane quarter + 4 x column group; a thread makes 8 columns of a chunk: the
//              epilogues are latency chains -- TMEM read, ex2, conversions -- and four warps per scheduler hide them
//              better than two: K3 321 -> 312 us on config 4): make the A operand of phases 1-7 in 32-wide K chunks (hi | lo, K-major,
//              SWIZZLE_64B) from the previous accumulator in TMEM (bias, CELU, CELU', Hadamard), and
//              drain g;
//   warp 16    TMA: streams the pre-packed, pre-swizzled weight chunks (hi | lo) of the schedule
//              from L2 into a 4-slot ring with cp.async.bulk + mbarrier;
//   warp 17    walks the MMA schedule; one elected lane issues tcgen05.mma and commits to the ring / phase barriers;
//   warp 18    TMA: the A operand of phase 0, which K2 writes in exactly the chunk image the tensor core reads
//              (AEV times 8, fp16 hi | lo, SWIZZLE_64B; one contiguous 16 KB block per tile and chunk), into the
//              3-slot ring A (its own thread: no head-of-line blocking behind the weight stream).
// Schedule.  The eight phases of a tile are a serial chain (each needs the previous
// accumulator), except at its two ends: the first GEMM (AEV x W1) depends only on global
// memory and the three g passes (delta1 x W1^T) only on delta1.  So consecutive tiles are
// software-pipelined: while the tensor pipe runs the g passes of tile t (delta1 kept RESIDENT in
// shared memory, produced once) it also runs the first GEMM of tile t+1 (the "overlapped
// block"); meanwhile warps 0-3 drain g of tile t (TMEM -> global, two accumulator buffers).  Then all
// sixteen worker warps walk the chain z1 -> h1 -> z2 -> h2 -> z3 -> delta3 -> d2pre -> delta2 -> d1pre -> delta1.
// TMEM (512 columns):  z1 [0,160)   z2 [160,288)   z3 [288,384)   d2pre [384,512)
//                      d1pre [160,320)   g buffer A [384,512)   g buffer B [160,288)
// The accumulate step of the tensor core rounds toward zero -- the running sum once per MMA
// instruction, and every product as it is aligned to it (measured: a chain of n K=16 MMAs shrinks
// an all-positive sum by 9e-8 n, a mixed-sign one by 2e-8 n); the one-sided loss is compensated in
// the epilogues: every phase returns (1 + beta_p) z with beta_p = lambda n_p 2.15e-8 (ks, kb below);
// lambda (forward phases / backward phases) is calibrated per element against the library's own
// FP32 MLP on the handle's first batch (pfc_api.cu: calibrate_tc).
#pragma once
#include <cuda_fp16.h>

#include "pfc_common.cuh"
#include "tc_ptx.cuh"

namespace pfc {

constexpr int TC_TM = 128;                       // rows per tile == ROW_PAD
constexpr int TC_CW = 8;                         // columns of a 32-wide chunk one worker thread makes (8 or 16)
constexpr int TC_NWW = 4 * (32 / TC_CW);         // worker warps: 4 TMEM lane quarters x column groups
constexpr int TC_WORKERS = 32 * TC_NWW;          // warps 0 .. TC_NWW-1
constexpr int TC_THREADS = TC_WORKERS + 96;      // + weight TMA warp, MMA warp, A-operand TMA warp
constexpr int TC_KC = 32;                        // k per chunk: one 64-byte SWIZZLE_64B row of fp16
constexpr int TC_NA = 3, TC_NB = 4;              // ring depths: A operand chunks, weight chunks
constexpr int TC_A_HALF = TC_TM * 64;            // 8,192 B: one part (hi or lo) of an A chunk
constexpr int TC_A_SLOT = 2 * TC_A_HALF;         // 16,384 B: hi | lo
constexpr int TC_B_SLOT = 2 * D1 * 64;           // 20,480 B: widest N (160), hi | lo
constexpr int TC_ND1 = D1 / TC_KC;               // 5 resident delta1 chunks
constexpr int TC_NPHASE = 8;
constexpr int TC_GN = 128;                       // g is produced in 3 passes of 128 columns
constexpr int TC_NPASS = D0 / TC_GN;             // 3
constexpr int TC_COL_Z1 = 0, TC_COL_Z2 = 160, TC_COL_Z3 = 288, TC_COL_D2 = 384, TC_COL_D1 = 160,
              TC_COL_GA = 384, TC_COL_GB = 160;
constexpr int TC_AEV_SCALE_LOG2 = 3;             // the AEV operand is multiplied by 8 before the split

// phase schedule: N, K chunks, packed-weight byte offset (per element)
//   0: W1 (N 160, K 384)   1: W2 (128, 160)   2: W3 (96, 128)   3: W3^T (128, 96)   4: W2^T (160, 128)
//   5-7: W1^T in three passes (128, 160)
__host__ __device__ constexpr int tc_phase_n(int p) {
  return p == 0 ? D1 : p == 1 ? D2 : p == 2 ? D3 : p == 3 ? D2 : p == 4 ? D1 : TC_GN;
}
__host__ __device__ constexpr int tc_phase_nk(int p) {
  return p == 0 ? D0 / TC_KC : p == 1 ? D1 / TC_KC : p == 2 ? D2 / TC_KC : p == 3 ? D3 / TC_KC : p == 4 ? D2 / TC_KC : D1 / TC_KC;
}
// MMA instructions of the accumulator chain of epilogue q (0..4: phases 0..4; 5: one g pass): 2 k steps per chunk
__host__ __device__ constexpr int tc_chain_mmas(int q, int n_terms) { return 2 * n_terms * tc_phase_nk(q); }
__host__ __device__ constexpr int tc_chunk_bytes(int p) { return 2 * tc_phase_n(p) * 64; }
__host__ __device__ constexpr int tc_phase_off(int p) {
  int o = 0;
  for (int q = 0; q < p; ++q) o += tc_phase_nk(q) * tc_chunk_bytes(q);
  return o;
}
constexpr int TC_W_BYTES_PER_ELEM = tc_phase_off(TC_NPHASE);        // 753,664
static_assert(TC_W_BYTES_PER_ELEM == 753664, "packed weight image");

// The overlapped block: 15 g-pass chunks of the previous tile and 12 first-GEMM chunks of the
// current one, in the fixed order the MMA issuer and the weight stream both follow.  Entry =
// kind << 8 | pass << 4 | chunk;  kind 0 = g pass (pass 0..2, chunk 0..4), kind 1 = first GEMM.
// Pass 0 runs first (its operand is ready when the block starts, the AEV chunks are still in
// flight); the first GEMM ends the block, so that the last drain overlaps its tail.
constexpr int TC_BLOCK_OPS = 27;
__host__ __device__ constexpr int tc_block_op(int i) {
  constexpr int G = 0, A = 1 << 8;
  const int t[TC_BLOCK_OPS] = {
      G | 0x00, G | 0x01, G | 0x02, G | 0x03, G | 0x04,
      A | 0, G | 0x10, A | 1, G | 0x11, A | 2, G | 0x12, A | 3, G | 0x13, A | 4, G | 0x14,
      A | 5, G | 0x20, A | 6, G | 0x21, A | 7, G | 0x22, A | 8, G | 0x23, G | 0x24,
      A | 9, A | 10, A | 11};
  return t[i];
}

struct TcSmem {                                   // after the 1024-aligned operand regions
  uint64_t a0_full[TC_NA], a_full[TC_NA], a_empty[TC_NA];   // ring A: first-GEMM chunks (bulk copy) / chain chunks (256 producers)
  uint64_t b_full[TC_NB], b_empty[TC_NB];
  uint64_t z_full[5];                             // accumulators z1, z2, z3, d2pre, d1pre complete
  uint64_t g_full[2];                             // g buffer A / B complete
  uint64_t g_free;                                // g buffer A drained (128 drain threads)
  uint64_t d1_full[TC_ND1];                       // resident delta1 chunk written (256)
  uint64_t d1_free;                               // every g-pass MMA of the tile has read the resident delta1
  uint64_t dd_full;                               // the four delta2 chunks are written to the resident region (256)
  uint64_t p5_done;                               // the delta1 producers have finished reading TMEM (256)
  uint32_t tmem_base;
  float4 stage[4][32 * 8];                        // per drain warp: 32 rows x 32 columns of g, 16-byte units XOR-swizzled by row
};
constexpr size_t TC_SMEM_BYTES = 1024 + (size_t)TC_ND1 * TC_A_SLOT + (size_t)TC_NA * TC_A_SLOT +
                                 (size_t)TC_NB * TC_B_SLOT + sizeof(TcSmem);
static_assert(TC_SMEM_BYTES <= 227 * 1024, "shared memory budget");

// per element: b1[160] b2[128] b3[96] w4[96] b4[1] pad[3] w4s[96] (w4 times the delta scale) ks[6] kb[6]
// Epilogue q returns ks[q] z + kb[q] z: ks[q] = 2^-(operand scales), an exact power of two, and
// kb[q] = beta_q ks[q] the truncation compensation -- two FMAs, because (1 + beta) itself is not
// representable finer than 1.2e-7 and beta_q is 4e-7 .. 1.5e-6.
constexpr int TC_BIAS_B1 = 0, TC_BIAS_B2 = D1, TC_BIAS_B3 = D1 + D2, TC_BIAS_W4 = D1 + D2 + D3,
              TC_BIAS_B4 = D1 + D2 + D3 + D3, TC_BIAS_W4S = 484, TC_BIAS_KS = 580, TC_BIAS_KB = 586, TC_BIAS_LEN = 592;

struct TcParams {
  const uint8_t* wpack;        // [NSPEC][TC_W_BYTES_PER_ELEM] packed hi|lo swizzled weight chunks (scaled)
  const float* bias[NSPEC];    // TC_BIAS_LEN floats per element (ks[q], kb[q]: scale and compensation of epilogue q)
  int row_start[NSPEC + 1];
  int n_tiles;
  long long* trace;            // DEVICE or NULL: pfc_k3_timeline (CTA 0 records clock64 at the events of TC_TRACE_*)
};

// ---- kind::f16 descriptors ----------------------------------------------------------------------
// Shared-memory matrix descriptor, K-major operand, SWIZZLE_64B: rows of 64 bytes (32 fp16),
// 8-row groups 512 bytes apart (SBO), 16-byte unit u of row r stored at unit u ^ ((r >> 1) & 3).
// [0,14) start>>4 | [16,30) LBO>>4 (=1, unused when swizzled) | [32,46) SBO>>4 |
// [46,48) version = 1 | [61,64) layout: 4 = SWIZZLE_64B.
__device__ __forceinline__ uint64_t tc_desc_sw64(uint32_t smem_addr) {
  uint64_t d = (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(512 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)4 << 61;
  return d;
}
// byte offset of fp16 element (row r, k in 0..31) inside a [rows x 32] SWIZZLE_64B tile
__host__ __device__ constexpr uint32_t tc_sw64_off(uint32_t r, uint32_t k) {
  return (r >> 3) * 512u + (r & 7u) * 64u + ((((k >> 3) ^ ((r >> 1) & 3u)) << 4) | ((k & 7u) << 1));
}
// Instruction descriptor, kind::f16, fp32 accumulate, fp16 A and B, both K-major, M x N tile:
// [4,6) D fmt: 1 = f32 | [7,10) A fmt: 0 = f16 | [10,13) B fmt: 0 = f16 | [15] A major: 0 = K |
// [16] B major: 0 = K | [17,23) N>>3 | [24,29) M>>4.
__host__ __device__ constexpr uint32_t tc_idesc_f16(int M, int N) {
  return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void tc_mma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}

// one lane of a converged warp (elect.sync: ptxas then knows that a single thread runs the guarded region and moves
// its operands to uniform registers without a waterfall loop)
__device__ __forceinline__ bool tc_elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}

// (x0, x1) -> packed (hi, lo): hi = fp16(x) to nearest, lo = fp16(x - hi) (x - hi is exact in fp32)
__device__ __forceinline__ void tc_split2(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(x0, x1);
  const float2 r = pk_fma(__half22float2(h), make_float2(-1.0f, -1.0f), make_float2(x0, x1));   // x - hi, both lanes
  const __half2 l = __floats2half2_rn(r.x, r.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// CELU(x) and CELU'(x), alpha = 0.1, branch-free:  e = exp(min(x,0)/alpha) is exactly 1 for x >= 0, so
//   CELU'(x) = e   and   CELU(x) = max(x,0) + alpha (e - 1)
__device__ __forceinline__ float celu_d(float x) { return ex2_approx(fminf(x, 0.0f) * (LOG2E / CELU_ALPHA)); }
__device__ __forceinline__ float celu_h(float x) { return fmaxf(x, 0.0f) + fmaf(CELU_ALPHA, celu_d(x), -CELU_ALPHA); }
__device__ __forceinline__ void celu_both(float x, float& h, float& d) {
  d = celu_d(x);
  h = fmaxf(x, 0.0f) + fmaf(CELU_ALPHA, d, -CELU_ALPHA);
}
// The epilogues work on PAIRS of columns in packed fp32 (fma.rn.f32x2 / mul.rn.f32x2: one issue slot for two lanes of
// arithmetic, same rounding as the scalar forms): they are bound by instruction issue (16 instructions per element
// in scalar form, two worker warps per scheduler), not by a pipe.
//   x = ks z + (kb z + b)   (operand scale, truncation compensation, bias)
__device__ __forceinline__ float2 tc_affine2(float z0, float z1, float2 ks, float2 kb, float b0, float b1) {
  const float2 z = make_float2(z0, z1);
  return pk_fma(z, ks, pk_fma(z, kb, make_float2(b0, b1)));
}
__device__ __forceinline__ float2 celu_d2(float2 x) {
  const float2 a = pk_mul(make_float2(fminf(x.x, 0.0f), fminf(x.y, 0.0f)), make_float2(LOG2E / CELU_ALPHA, LOG2E / CELU_ALPHA));
  return make_float2(ex2_approx(a.x), ex2_approx(a.y));
}
__device__ __forceinline__ float2 celu_h2(float2 x, float2 d) {
  const float2 t = pk_fma(make_float2(CELU_ALPHA, CELU_ALPHA), d, make_float2(-CELU_ALPHA, -CELU_ALPHA));
  return pk_fma(make_float2(fmaxf(x.x, 0.0f), fmaxf(x.y, 0.0f)), make_float2(1.0f, 1.0f), t);
}

// TC_CW consecutive floats of an aligned table (biases, w4) through the read-only path, 16-byte loads
__device__ __forceinline__ void tc_ldw(const float* p, float (&v)[TC_CW]) {
#pragma unroll
  for (int j = 0; j < TC_CW / 4; ++j) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p) + j);
    v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
  }
}
// my accumulator columns TMEM -> registers (8 or 16 per thread)
__device__ __forceinline__ void tc_tmem_ldw(uint32_t taddr, float (&v)[16]) { tc::tmem_ld16(taddr, v); }
__device__ __forceinline__ void tc_tmem_ldw(uint32_t taddr, float (&v)[8]) { tc::tmem_ld8(taddr, v); }
// store TC_CW consecutive K values (columns TC_CW*hf .. of a 32-wide chunk) of row r as hi | lo
__device__ __forceinline__ void tc_store_aw(uint8_t* slot, int r, int hf, const float (&v)[TC_CW]) {
  uint32_t hi[TC_CW / 2], lo[TC_CW / 2];
#pragma unroll
  for (int j = 0; j < TC_CW / 2; ++j) tc_split2(v[2 * j], v[2 * j + 1], hi[j], lo[j]);
  const uint32_t row = (uint32_t)(r >> 3) * 512u + (uint32_t)(r & 7) * 64u, sw = (uint32_t)(r >> 1) & 3u;
#pragma unroll
  for (int u = 0; u < TC_CW / 8; ++u) {
    const uint32_t off = row + ((((uint32_t)((TC_CW / 8) * hf + u)) ^ sw) << 4);
    *reinterpret_cast<uint4*>(slot + off) = make_uint4(hi[4 * u], hi[4 * u + 1], hi[4 * u + 2], hi[4 * u + 3]);
    *reinterpret_cast<uint4*>(slot + TC_A_HALF + off) = make_uint4(lo[4 * u], lo[4 * u + 1], lo[4 * u + 2], lo[4 * u + 3]);
  }
}

// pfc_k3_timeline: 64 slots per tile iteration of CTA 0.  MMA issuer: 0 iteration start, 1..27 after block op i,
// 28..31 after the chain GEMMs 1..4 are issued.  Worker thread 0 (drain group): 32 block start, 33..35 after drain
// pass 0..2, then 36/37 .. 44/45 = accumulator seen / operand written for h1, h2, delta3, delta2, delta1.  Worker
// (slots 48.. unused).
constexpr int TC_TRACE_STRIDE = 128, TC_TRACE_ITERS = 8;
#define TC_TRACE(slot)                                                                              \
  do {                                                                                              \
    if (P.trace != nullptr && blockIdx.x == 0 && it < TC_TRACE_ITERS) P.trace[it * TC_TRACE_STRIDE + (slot)] = clock64(); \
  } while (0)

template <int N_TERMS>
__global__ void __launch_bounds__(TC_THREADS, 1)
k3_mlp_tc_kernel(const __grid_constant__ TcParams P, const uint8_t* __restrict__ aev16, float* __restrict__ g,
                 float* __restrict__ e_row) {
  extern __shared__ uint8_t smem_raw[];
  // 1024-byte alignment by pointer arithmetic on the shared array (an integer round trip would turn every
  // access below into a generic load / store)
  uint8_t* base = smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u);
  uint8_t* resD1 = base;                                   // resident delta1 operand: 5 chunks
  uint8_t* ringA = resD1 + TC_ND1 * TC_A_SLOT;
  uint8_t* ringB = ringA + TC_NA * TC_A_SLOT;
  TcSmem& S = *reinterpret_cast<TcSmem*>(ringB + TC_NB * TC_B_SLOT);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int i = 0; i < TC_NA; ++i) {
      tc::mbar_init(&S.a0_full[i], 1); tc::mbar_init(&S.a_full[i], TC_WORKERS); tc::mbar_init(&S.a_empty[i], 1);
    }
    for (int i = 0; i < TC_NB; ++i) { tc::mbar_init(&S.b_full[i], 1); tc::mbar_init(&S.b_empty[i], 1); }
    for (int i = 0; i < 5; ++i) tc::mbar_init(&S.z_full[i], 1);
    tc::mbar_init(&S.g_full[0], 1); tc::mbar_init(&S.g_full[1], 1);
    tc::mbar_init(&S.g_free, 128);
    for (int i = 0; i < TC_ND1; ++i) tc::mbar_init(&S.d1_full[i], TC_WORKERS);
    tc::mbar_init(&S.d1_free, 1);
    tc::mbar_init(&S.dd_full, TC_WORKERS);
    tc::mbar_init(&S.p5_done, TC_WORKERS);
    tc::mbar_fence_init();
  }
  if (warp == TC_NWW + 1) tc::tmem_alloc<512>(&S.tmem_base);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tbase = S.tmem_base;
  // tiles of this CTA: blockIdx.x, blockIdx.x + gridDim.x, ...; iteration `it` runs the overlapped block of
  // (tile it-1, tile it) and then the chain of tile it; one extra iteration drains the last tile
  const int n_my = (P.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  auto tile_of = [&](int it) { return (int)blockIdx.x + it * (int)gridDim.x; };
  auto elem_of = [&](int tile) {
    int el = 0;
#pragma unroll
    for (int k = 1; k < NSPEC; ++k) el += (tile * TC_TM >= P.row_start[k]);
    return el;
  };

  if (warp < TC_NWW) {
    // =========================== workers ===========================
    const int q = warp & 3, hf = warp >> 2;
    const int r = 32 * q + lane;                               // tile row == TMEM lane
    const uint32_t tlane = tbase + ((uint32_t)(32 * q) << 16);
    uint32_t ia = 0;                                           // ring A chunks so far (all kinds)
    auto acquire = [&]() -> uint8_t* {                         // wait until slot ia % NA is free
      const uint32_t s = ia % TC_NA, use = ia / TC_NA;
      tc::mbar_wait(&S.a_empty[s], (use & 1u) ^ 1u);
      return ringA + s * TC_A_SLOT;
    };
    auto publish = [&](uint64_t* bar) {
      tc::tc_fence_before();                                   // this thread's tcgen05.ld precede the MMAs that overwrite
      tc::fence_proxy_async_smem();
      tc::mbar_arrive(bar);
    };
    for (int it = 0; it <= n_my; ++it) {
      const bool have_prev = it >= 1, have_cur = it < n_my;
      const uint32_t par = (uint32_t)it & 1u, par_prev = ((uint32_t)it + 1u) & 1u;
      if (tid == 0) TC_TRACE(32);
      // ------------------------------ overlapped block ------------------------------
      if (hf == 0) {
        // drain g of the previous tile: pass 0 and 2 from buffer A, pass 1 from buffer B
        if (have_prev) {
          const int row0 = tile_of(it - 1) * TC_TM;
          const float* bprev = P.bias[elem_of(tile_of(it - 1))];
          const float kg = __ldg(bprev + TC_BIAS_KS + 5), kgb = __ldg(bprev + TC_BIAS_KB + 5);
#pragma unroll 1
          for (int pass = 0; pass < TC_NPASS; ++pass) {
            const int buf = pass == 1 ? 1 : 0;
            // completions of g_full[A]: two per tile (2(it-1), 2(it-1)+1); of g_full[B]: one per tile
            tc::mbar_wait(&S.g_full[buf], buf ? par_prev : (uint32_t)(pass >> 1));
            tc::tc_fence_after();
            const uint32_t col = (uint32_t)(buf ? TC_COL_GB : TC_COL_GA);
            // 32 x 32 blocks: TMEM gives every lane its own row; the block is transposed through shared
            // memory so that each store instruction writes four complete 128-byte row segments (a lane
            // storing its own row touched 32 different lines per instruction: 3.7 us per pass, measured)
            float4* stg = S.stage[q];
#pragma unroll 1
            for (int c = 0; c < TC_GN / 32; ++c) {
              float v0[16], v1[16];
              tc::tmem_ld16(tlane + col + 32 * c, v0);
              tc::tmem_ld16(tlane + col + 32 * c + 16, v1);
              tc::tmem_ld_wait();
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                auto sc2 = [&](float a, float b) {
                  const float2 v = make_float2(a, b);
                  return pk_fma(v, make_float2(kgb, kgb), pk_mul(v, make_float2(kg, kg)));
                };
                const float2 a0 = sc2(v0[4 * k], v0[4 * k + 1]), a1 = sc2(v0[4 * k + 2], v0[4 * k + 3]);
                const float2 b0 = sc2(v1[4 * k], v1[4 * k + 1]), b1 = sc2(v1[4 * k + 2], v1[4 * k + 3]);
                stg[lane * 8 + (k ^ (lane & 7))] = make_float4(a0.x, a0.y, a1.x, a1.y);
                stg[lane * 8 + ((4 + k) ^ (lane & 7))] = make_float4(b0.x, b0.y, b1.x, b1.y);
              }
              __syncwarp();
              float* blk = g + (size_t)(row0 + 32 * q) * AEV_LEN + pass * TC_GN + 32 * c;
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const int rr = 4 * i + (lane >> 3), u = lane & 7;
                *reinterpret_cast<float4*>(blk + (size_t)rr * AEV_LEN + 4 * u) = stg[rr * 8 + (u ^ (rr & 7))];
              }
              __syncwarp();
            }
            if (buf == 0) {
              tc::tc_fence_before();
              tc::mbar_arrive(&S.g_free);
            }
            if (tid == 0) TC_TRACE(33 + pass);
          }
        }
      }
      if (have_cur) ia += D0 / TC_KC;                          // the twelve first-GEMM chunks come by bulk copy (warp 18)
      if (!have_cur) break;
      // ------------------------------ chain of the current tile ------------------------------
      const int row0 = tile_of(it) * TC_TM;
      const float* bias = P.bias[elem_of(tile_of(it))];
      const float k0 = __ldg(bias + TC_BIAS_KS + 0), k1 = __ldg(bias + TC_BIAS_KS + 1), k2 = __ldg(bias + TC_BIAS_KS + 2),
                  k3 = __ldg(bias + TC_BIAS_KS + 3), k4 = __ldg(bias + TC_BIAS_KS + 4);
      const float c0 = __ldg(bias + TC_BIAS_KB + 0), c1 = __ldg(bias + TC_BIAS_KB + 1), c2 = __ldg(bias + TC_BIAS_KB + 2),
                  c3 = __ldg(bias + TC_BIAS_KB + 3), c4 = __ldg(bias + TC_BIAS_KB + 4);
      const float2 ks0 = make_float2(k0, k0), ks1 = make_float2(k1, k1), ks2 = make_float2(k2, k2), ks3 = make_float2(k3, k3),
                   ks4 = make_float2(k4, k4), kb0 = make_float2(c0, c0), kb1 = make_float2(c1, c1), kb2 = make_float2(c2, c2),
                   kb3 = make_float2(c3, c3), kb4 = make_float2(c4, c4);
      // ---- z1 -> h1 = CELU(z1 + b1): operand of phase 1 ----
      tc::mbar_wait(&S.z_full[0], par);
      tc::tc_fence_after();
      if (tid == 0) TC_TRACE(36);
#pragma unroll 1
      for (int c = 0; c < D1 / TC_KC; ++c) {
        float z[TC_CW], h[TC_CW];
        tc_tmem_ldw(tlane + TC_COL_Z1 + 32 * c + TC_CW * hf, z);
        tc::tmem_ld_wait();
        float bb[TC_CW];
        tc_ldw(bias + TC_BIAS_B1 + 32 * c + TC_CW * hf, bb);
#pragma unroll
        for (int k = 0; k < TC_CW; k += 2) {
          const float2 x = tc_affine2(z[k], z[k + 1], ks0, kb0, bb[k], bb[k + 1]);
          const float2 hh = celu_h2(x, celu_d2(x));
          h[k] = hh.x; h[k + 1] = hh.y;
        }
        uint8_t* slot = acquire();
        tc_store_aw(slot, r, hf, h);
        publish(&S.a_full[ia % TC_NA]);
        ++ia;
      }
      if (tid == 0) TC_TRACE(37);
      // ---- z2 -> h2: operand of phase 2 ----
      tc::mbar_wait(&S.z_full[1], par);
      tc::tc_fence_after();
      if (tid == 0) TC_TRACE(38);
#pragma unroll 1
      for (int c = 0; c < D2 / TC_KC; ++c) {
        float z[TC_CW], h[TC_CW];
        tc_tmem_ldw(tlane + TC_COL_Z2 + 32 * c + TC_CW * hf, z);
        tc::tmem_ld_wait();
        float bb[TC_CW];
        tc_ldw(bias + TC_BIAS_B2 + 32 * c + TC_CW * hf, bb);
#pragma unroll
        for (int k = 0; k < TC_CW; k += 2) {
          const float2 x = tc_affine2(z[k], z[k + 1], ks1, kb1, bb[k], bb[k + 1]);
          const float2 hh = celu_h2(x, celu_d2(x));
          h[k] = hh.x; h[k + 1] = hh.y;
        }
        uint8_t* slot = acquire();
        tc_store_aw(slot, r, hf, h);
        publish(&S.a_full[ia % TC_NA]);
        ++ia;
      }
      if (tid == 0) TC_TRACE(39);
      // ---- z3 -> e_i = w4.h3 + b4 and delta3 = w4 * CELU'(z3 + b3) (scaled): operand of phase 3 ----
      tc::mbar_wait(&S.z_full[2], par);
      tc::tc_fence_after();
      if (tid == 0) TC_TRACE(40);
      {
        float2 epart2 = make_float2(0.0f, 0.0f);            // even / odd columns, added at the end
#pragma unroll 1
        for (int c = 0; c < D3 / TC_KC; ++c) {
          float z[TC_CW], dl[TC_CW];
          tc_tmem_ldw(tlane + TC_COL_Z3 + 32 * c + TC_CW * hf, z);
          tc::tmem_ld_wait();
          float bb[TC_CW], w4[TC_CW], w4s[TC_CW];
          tc_ldw(bias + TC_BIAS_B3 + 32 * c + TC_CW * hf, bb);
          tc_ldw(bias + TC_BIAS_W4 + 32 * c + TC_CW * hf, w4);
          tc_ldw(bias + TC_BIAS_W4S + 32 * c + TC_CW * hf, w4s);
#pragma unroll
          for (int k = 0; k < TC_CW; k += 2) {
            const float2 x = tc_affine2(z[k], z[k + 1], ks2, kb2, bb[k], bb[k + 1]);
            const float2 d = celu_d2(x);
            epart2 = pk_fma(make_float2(w4[k], w4[k + 1]), celu_h2(x, d), epart2);
            const float2 dd = pk_mul(make_float2(w4s[k], w4s[k + 1]), d);
            dl[k] = dd.x; dl[k + 1] = dd.y;
          }
          uint8_t* slot = acquire();
          tc_store_aw(slot, r, hf, dl);
          publish(&S.a_full[ia % TC_NA]);
          ++ia;
        }
        // (energy partials share the drain's staging block: every drain of the previous tile is over before z3 exists,
        // and the next drain starts behind the barrier below)
        float (*epart)[TC_TM] = reinterpret_cast<float (*)[TC_TM]>(&S.stage[0][0]);
        epart[hf][r] = epart2.x + epart2.y;
        asm volatile("bar.sync 1, %0;" ::"n"(TC_WORKERS) : "memory");
        if (hf == 0) {
          float es = epart[0][r];
#pragma unroll
          for (int k = 1; k < 32 / TC_CW; ++k) es += epart[k][r];
          e_row[row0 + r] = es + __ldg(bias + TC_BIAS_B4);
        }
      }
      if (tid == 0) TC_TRACE(41);
      // ---- delta2 = d2pre * CELU'(z2 + b2): operand of phase 4 ----
      // d1pre (phase 4's accumulator) overwrites z2 / z3, so phase 4 cannot start before ALL of delta2
      // exists: its four chunks go to the resident region (free at this point: the previous tile's g
      // passes are over), not through the three-slot ring, which could not hold them
      tc::mbar_wait(&S.z_full[3], par);
      tc::tc_fence_after();
      if (tid == 0) TC_TRACE(42);
      if (have_prev) tc::mbar_wait(&S.d1_free, par_prev);      // the previous tile's g passes have read the region
#pragma unroll 1
      for (int c = 0; c < D2 / TC_KC; ++c) {
        float z[TC_CW], p[TC_CW];
        tc_tmem_ldw(tlane + TC_COL_Z2 + 32 * c + TC_CW * hf, z);
        tc_tmem_ldw(tlane + TC_COL_D2 + 32 * c + TC_CW * hf, p);
        tc::tmem_ld_wait();
        float bb[TC_CW];
        tc_ldw(bias + TC_BIAS_B2 + 32 * c + TC_CW * hf, bb);
#pragma unroll
        for (int k = 0; k < TC_CW; k += 2) {
          const float2 pp = make_float2(p[k], p[k + 1]);
          const float2 t = pk_mul(pk_fma(pp, kb3, pk_mul(pp, ks3)), celu_d2(tc_affine2(z[k], z[k + 1], ks1, kb1, bb[k], bb[k + 1])));
          p[k] = t.x; p[k + 1] = t.y;
        }
        tc_store_aw(resD1 + c * TC_A_SLOT, r, hf, p);
      }
      publish(&S.dd_full);
      if (tid == 0) TC_TRACE(43);
      // ---- delta1 = d1pre * CELU'(z1 + b1): RESIDENT operand of the three g passes ----
      tc::mbar_wait(&S.z_full[4], par);                        // (phase 4 has consumed delta2: the region is free again)
      tc::tc_fence_after();
      if (tid == 0) TC_TRACE(44);
#pragma unroll 1
      for (int c = 0; c < TC_ND1; ++c) {
        float z[TC_CW], p[TC_CW];
        tc_tmem_ldw(tlane + TC_COL_Z1 + 32 * c + TC_CW * hf, z);
        tc_tmem_ldw(tlane + TC_COL_D1 + 32 * c + TC_CW * hf, p);
        tc::tmem_ld_wait();
        float bb[TC_CW];
        tc_ldw(bias + TC_BIAS_B1 + 32 * c + TC_CW * hf, bb);
#pragma unroll
        for (int k = 0; k < TC_CW; k += 2) {
          const float2 pp = make_float2(p[k], p[k + 1]);
          const float2 t = pk_mul(pk_fma(pp, kb4, pk_mul(pp, ks4)), celu_d2(tc_affine2(z[k], z[k + 1], ks0, kb0, bb[k], bb[k + 1])));
          p[k] = t.x; p[k + 1] = t.y;
        }
        tc_store_aw(resD1 + c * TC_A_SLOT, r, hf, p);
        publish(&S.d1_full[c]);
      }
      tc::tc_fence_before();
      tc::mbar_arrive(&S.p5_done);
      if (tid == 0) TC_TRACE(45);
    }
  } else if (warp == TC_NWW) {
    // =========================== TMA: weight chunks ===========================
    if (lane == 0) {
      uint32_t ib = 0;
      auto stream = [&](const uint8_t* src, uint32_t bytes) {
        const uint32_t s = ib % TC_NB, use = ib / TC_NB;
        tc::mbar_wait(&S.b_empty[s], (use & 1u) ^ 1u);
        tc::mbar_arrive_expect_tx(&S.b_full[s], bytes);
        tc::bulk_g2s(ringB + s * TC_B_SLOT, src, bytes, &S.b_full[s]);
        ++ib;
      };
      for (int it = 0; it <= n_my; ++it) {
        const bool have_prev = it >= 1, have_cur = it < n_my;
        const uint8_t* wprev = have_prev ? P.wpack + (size_t)elem_of(tile_of(it - 1)) * TC_W_BYTES_PER_ELEM : nullptr;
        const uint8_t* wcur = have_cur ? P.wpack + (size_t)elem_of(tile_of(it)) * TC_W_BYTES_PER_ELEM : nullptr;
#pragma unroll 1
        for (int i = 0; i < TC_BLOCK_OPS; ++i) {
          const int op = tc_block_op(i);
          if (op >> 8) {
            if (have_cur) stream(wcur + tc_phase_off(0) + (size_t)(op & 15) * tc_chunk_bytes(0), (uint32_t)tc_chunk_bytes(0));
          } else if (have_prev) {
            stream(wprev + tc_phase_off(5 + ((op >> 4) & 3)) + (size_t)(op & 15) * tc_chunk_bytes(5), (uint32_t)tc_chunk_bytes(5));
          }
        }
        if (!have_cur) break;
#pragma unroll 1
        for (int p = 1; p <= 4; ++p) {
          const uint8_t* src = wcur + tc_phase_off(p);
          const uint32_t bytes = (uint32_t)tc_chunk_bytes(p);
          for (int c = 0; c < tc_phase_nk(p); ++c) stream(src + (size_t)c * bytes, bytes);
        }
      }
    }
  } else if (warp == TC_NWW + 2) {
    // =========================== TMA: the first GEMM's A operand ===========================
    // its own thread, so that a chunk is requested the moment a ring-A slot frees (up to three chunks ahead, and
    // already during the previous tile's last epilogues) instead of when the weight stream's walk reaches it
    if (lane == 0) {
      uint32_t ia = 0, par_a1 = 0;
      for (int it = 0; it < n_my; ++it) {
        const uint8_t* src = aev16 + (size_t)tile_of(it) * (D0 / TC_KC) * TC_A_SLOT;
#pragma unroll 1
        for (int c = 0; c < D0 / TC_KC; ++c) {                 // (hi | lo chunk image, as K2 wrote it)
          const uint32_t s = ia % TC_NA, use = ia / TC_NA;
          tc::mbar_wait(&S.a_empty[s], (use & 1u) ^ 1u);
          tc::mbar_arrive_expect_tx(&S.a0_full[s], (uint32_t)TC_A_SLOT);
          tc::bulk_g2s(ringA + s * TC_A_SLOT, src + (size_t)c * TC_A_SLOT, (uint32_t)TC_A_SLOT, &S.a0_full[s]);
          ++ia;
        }
        // the chain's twelve ring-A chunks are made by the workers.  This thread follows their production (a_full)
        // before it asks for a slot again: a parity wait on a_empty cannot tell the completion it needs from one
        // several uses earlier, so it must never be more than one use of a slot ahead
#pragma unroll 1
        for (int c = 0; c < tc_phase_nk(1) + tc_phase_nk(2) + tc_phase_nk(3); ++c) {
          const uint32_t s = ia % TC_NA;
          tc::mbar_wait(&S.a_full[s], (par_a1 >> s) & 1u);
          par_a1 ^= 1u << s;
          ++ia;
        }
      }
    }
  } else {
    // =========================== MMA issuer ===========================
    // The WHOLE warp walks the schedule with warp-uniform control flow and operands (ring counters, shared-memory
    // addresses, the TMEM base taken through a shuffle), so that descriptors and addresses are computed on the
    // uniform datapath; one elected lane issues the tcgen05.mma / commit instructions.  (With the walk inside `if (lane == 0)`
    // every MMA was wrapped in an ELECT / R2UR waterfall loop and the issuing thread, not the tensor pipe, paced the
    // overlapped block: 0.5 us per 32-k chunk against 0.3 us of MMA time, pfc_k3_timeline.)
    {
      const uint32_t tbase = __shfl_sync(0xffffffffu, S.tmem_base, 0);
      uint32_t ia = 0, ib = 0;
      uint32_t par_a0 = 0, par_a1 = 0;                         // per-slot phase parities of a0_full / a_full
      // one 32-k chunk: 2 k steps x N_TERMS MMAs of M 128 x N into TMEM column dcol; A from `a_slot`, B from ring slot
      auto issue = [&](uint32_t dcol, uint32_t a_slot, int N, bool first) {
        const uint32_t sb = ib % TC_NB;
        tc::mbar_wait(&S.b_full[sb], (ib / TC_NB) & 1u);
        tc::tc_fence_after();
        const uint32_t a_hi = a_slot, a_lo = a_slot + TC_A_HALF;
        const uint32_t b_hi = tc::smem_u32(ringB + sb * TC_B_SLOT), b_lo = b_hi + (uint32_t)N * 64u;
        const uint32_t idesc = tc_idesc_f16(TC_TM, N);
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
          const uint64_t dah = tc_desc_sw64(a_hi + 32 * ks), dal = tc_desc_sw64(a_lo + 32 * ks);
          const uint64_t dbh = tc_desc_sw64(b_hi + 32 * ks), dbl = tc_desc_sw64(b_lo + 32 * ks);
          if (tc_elect_one()) {
            if (N_TERMS == 3) {
              tc_mma_f16(dcol, dal, dbh, idesc, (first && ks == 0) ? 0u : 1u);
              tc_mma_f16(dcol, dah, dbl, idesc, 1u);
              tc_mma_f16(dcol, dah, dbh, idesc, 1u);
            } else {
              tc_mma_f16(dcol, dah, dbh, idesc, (first && ks == 0) ? 0u : 1u);
            }
          }
        }
        if (tc_elect_one()) tc::mma_commit(&S.b_empty[sb]);
        __syncwarp();
        ++ib;
      };
      // a chunk whose A operand comes through ring A (kind 0: first GEMM, bulk copy; kind 1: chain, 256 producers)
      auto issue_ring = [&](uint32_t dcol, int N, bool first, int kind) {
        const uint32_t sa = ia % TC_NA;
        if (kind == 0) { tc::mbar_wait(&S.a0_full[sa], (par_a0 >> sa) & 1u); par_a0 ^= 1u << sa; }
        else           { tc::mbar_wait(&S.a_full[sa], (par_a1 >> sa) & 1u); par_a1 ^= 1u << sa; }
        issue(dcol, tc::smem_u32(ringA + sa * TC_A_SLOT), N, first);
        if (tc_elect_one()) tc::mma_commit(&S.a_empty[sa]);
        ++ia;
      };
      for (int it = 0; it <= n_my; ++it) {
        const bool have_prev = it >= 1, have_cur = it < n_my;
        const uint32_t par_prev = ((uint32_t)it + 1u) & 1u;
        if (tc_elect_one()) TC_TRACE(0);
        // ------------------------------ overlapped block ------------------------------
        bool p5_waited = !have_prev;
#pragma unroll
        for (int i = 0; i < TC_BLOCK_OPS; ++i) {                  // (unrolled: the op table folds into constants)
          const int op = tc_block_op(i), c = op & 15;
          if (op >> 8) {                                       // first GEMM of the current tile -> z1
            if (!have_cur) continue;
            if (!p5_waited) { tc::mbar_wait(&S.p5_done, par_prev); p5_waited = true; }   // z1 / d1pre of the previous tile were read
            issue_ring(tbase + TC_COL_Z1, D1, c == 0, 0);
            if (c == D0 / TC_KC - 1 && tc_elect_one()) tc::mma_commit(&S.z_full[0]);
          } else {                                             // g pass of the previous tile
            if (!have_prev) continue;
            const int pass = (op >> 4) & 3;
            if (c == 0) {
              if (pass == 1 && !p5_waited) { tc::mbar_wait(&S.p5_done, par_prev); p5_waited = true; }   // buffer B = d1pre's columns
              if (pass == 2) tc::mbar_wait(&S.g_free, 0u);     // buffer A drained of pass 0 (completion 2(it-1))
            }
            if (pass == 0) tc::mbar_wait(&S.d1_full[c], par_prev);
            issue(tbase + (uint32_t)(pass == 1 ? TC_COL_GB : TC_COL_GA), tc::smem_u32(resD1 + c * TC_A_SLOT), TC_GN, c == 0);
            if (c == TC_ND1 - 1 && tc_elect_one()) {
              tc::mma_commit(&S.g_full[pass == 1 ? 1 : 0]);
              if (pass == TC_NPASS - 1) tc::mma_commit(&S.d1_free);
            }
          }
          if (tc_elect_one()) TC_TRACE(1 + i);
        }
        if (!have_cur) break;
        // ------------------------------ chain ------------------------------
        for (int c = 0; c < tc_phase_nk(1); ++c) issue_ring(tbase + TC_COL_Z2, tc_phase_n(1), c == 0, 1);
        if (tc_elect_one()) { tc::mma_commit(&S.z_full[1]); TC_TRACE(28); }
        for (int c = 0; c < tc_phase_nk(2); ++c) issue_ring(tbase + TC_COL_Z3, tc_phase_n(2), c == 0, 1);
        if (tc_elect_one()) { tc::mma_commit(&S.z_full[2]); TC_TRACE(29); }
        for (int c = 0; c < tc_phase_nk(3); ++c) issue_ring(tbase + TC_COL_D2, tc_phase_n(3), c == 0, 1);
        if (tc_elect_one()) { tc::mma_commit(&S.z_full[3]); TC_TRACE(30); }
        tc::mbar_wait(&S.dd_full, (uint32_t)it & 1u);            // all of delta2 is in the resident region
        for (int c = 0; c < tc_phase_nk(4); ++c)
          issue(tbase + TC_COL_D1, tc::smem_u32(resD1 + c * TC_A_SLOT), tc_phase_n(4), c == 0);
        if (tc_elect_one()) { tc::mma_commit(&S.z_full[4]); TC_TRACE(31); }
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == TC_NWW + 1) tc::tmem_dealloc<512>(tbase);
}

}  // namespace pfc
