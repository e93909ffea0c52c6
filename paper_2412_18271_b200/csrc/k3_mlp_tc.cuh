// k3_mlp_tc.cuh -- K3 (tensor-core path): the per-element MLP 384->160->128->96->1, forward and
// input-gradient backward, as a chain of eight grouped-GEMM phases per 128-row tile on the
// tcgen05 tensor cores (O5 / section 5; backward = PAPER.md:67 "forces by backprop").
//
// Precision: kind::tf32 with the 3-term split  A*B ~= A_hi*B_hi + A_lo*B_hi + A_hi*B_lo
// (x_hi = x rounded to 10 mantissa bits, x_lo = x - x_hi exactly), fp32 accumulation in TMEM.
// The hardware truncates fp32 operands to tf32 (measured), so every hi part is exact and the
// dropped terms are O(2^-21) relative.  N_TERMS = 1 is plain TF32, kept only to produce the
// evidence that it misses the tolerance.
//
// One persistent CTA per SM, 320 threads, one 128-row tile of ONE element in flight:
//   warps 0-7  producers/epilogue: make the A operand of every phase in 32-wide K chunks
//              (hi|lo, K-major, SWIZZLE_128B) into a 4-slot shared-memory ring -- phase 0 from
//              the AEV rows in global memory, later phases from the previous accumulator in
//              TMEM (bias, CELU, CELU', Hadamard) -- and drain g to global memory;
//   warp 8     TMA: streams the pre-packed, pre-swizzled weight chunks (hi|lo) of the phase
//              schedule from L2 into a 2-slot ring with cp.async.bulk + mbarrier;
//   warp 9     one elected thread issues tcgen05.mma and commits to the ring / phase barriers.
// TMEM (512 columns) keeps the forward pre-activations z1,z2,z3 for the backward pass:
//   z1 [0,160)  z2 [160,288)  z3 [288,384)  d2pre [384,512)  d1pre [160,320)  g-pass [384,512)
// The accumulate step of the tensor core rounds toward zero (measured: the energy error of a
// single-accumulator split correlates at -0.7 with the energy), one truncation per MMA, so the
// small terms A_lo*B_hi + A_hi*B_lo of phases 0 and 2 go to an accumulator of their own
// (S0 [352,512), S2 [384,480): free at that time) and are added on the CUDA cores; z1 is written
// back (bias included) for the backward pass.
// What remains of that one-sided loss is compensated in the epilogues: a chain of n MMA instructions
// shrinks its sum by a relative beta ~ lambda * n * 2.15e-8 on average (half an ulp of the running sum
// per step), so every phase returns z + beta_p * z (TcParams::comp; lambda measured against the fp64
// oracle).  With it the path meets the 1e-4 A trajectory bar on all five
// configurations and is what PFC_MLP_AUTO selects for batches of >= 4096 atoms.
#pragma once
#include "pfc_common.cuh"
#include "tc_ptx.cuh"

namespace pfc {

constexpr int TC_TM = 128;                       // rows per tile == ROW_PAD
constexpr int TC_THREADS = 320;
constexpr int TC_EPI_THREADS = 256;
constexpr int TC_NA = 4, TC_NB = 2;              // ring depths
constexpr int TC_A_SLOT = 2 * TC_TM * 128;       // 32,768 B: hi | lo
constexpr int TC_B_SLOT = 2 * D1 * 128;          // 40,960 B: widest N (160) hi | lo
constexpr int TC_NPHASE = 8;
constexpr int TC_GN = 128;                       // g is produced in 3 passes of 128 columns
constexpr int TC_S0_COL = 352, TC_S2_COL = 384;  // small-term accumulators of phases 0 and 2

// phase schedule: N, K chunks, D column, packed-weight byte offset (per element)
__host__ __device__ constexpr int tc_phase_n(int p) {
  return p == 0 ? D1 : p == 1 ? D2 : p == 2 ? D3 : p == 3 ? D2 : p == 4 ? D1 : TC_GN;
}
__host__ __device__ constexpr int tc_phase_nk(int p) {
  return p == 0 ? D0 / 32 : p == 1 ? D1 / 32 : p == 2 ? D2 / 32 : p == 3 ? D3 / 32 : p == 4 ? D2 / 32 : D1 / 32;
}
__host__ __device__ constexpr int tc_phase_dcol(int p) {
  return p == 0 ? 0 : p == 1 ? 160 : p == 2 ? 288 : p == 3 ? 384 : p == 4 ? 160 : 384;
}
__host__ __device__ constexpr int tc_chunk_bytes(int p) { return 2 * tc_phase_n(p) * 128; }
__host__ __device__ constexpr int tc_phase_off(int p) {
  int o = 0;
  for (int q = 0; q < p; ++q) o += tc_phase_nk(q) * tc_chunk_bytes(q);
  return o;
}
constexpr int TC_W_BYTES_PER_ELEM = tc_phase_off(TC_NPHASE);        // 1,507,328
constexpr int TC_CHUNKS_PER_TILE = 12 + 5 + 4 + 3 + 4 + 15;         // 43
static_assert(TC_W_BYTES_PER_ELEM == 1507328, "packed weight image");

struct TcSmem {                                   // after the 1024-aligned rings
  uint64_t a_full[TC_NA], a_empty[TC_NA], b_full[TC_NB], b_empty[TC_NB];
  uint64_t d_full, dg_free;
  uint32_t tmem_base;
  float epart[2][TC_TM];
};
constexpr size_t TC_SMEM_BYTES = 1024 + (size_t)TC_NA * TC_A_SLOT + (size_t)TC_NB * TC_B_SLOT + sizeof(TcSmem);

struct TcParams {
  const uint8_t* wpack;        // [NSPEC][TC_W_BYTES_PER_ELEM] packed hi|lo swizzled weight chunks
  const float* bias[NSPEC];    // per element: b1[160] b2[128] b3[96] w4[96] b4[1]  (481 floats)
  int row_start[NSPEC + 1];
  int n_tiles;
  float comp[6];               // expected relative truncation loss of the accumulator chain of phases 0..4 and the g passes
};
constexpr int TC_BIAS_B1 = 0, TC_BIAS_B2 = D1, TC_BIAS_B3 = D1 + D2, TC_BIAS_W4 = D1 + D2 + D3,
              TC_BIAS_B4 = D1 + D2 + D3 + D3, TC_BIAS_LEN = 484;

// x -> (hi, lo): hi = x rounded to tf32 precision (10 mantissa bits); lo = x - hi (exact in fp32)
// rounded to tf32 as well -- the tensor core would otherwise TRUNCATE it, a one-sided 2^-21 error
// that adds up linearly over K and over the atoms of a system; rounded, it is 2^-22 and unbiased.
__device__ __forceinline__ float tf32_round(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u);
}
__device__ __forceinline__ void tf32_split(float x, float& hi, float& lo) {
  hi = tf32_round(x);
  lo = tf32_round(x - hi);
}

// CELU(x) and CELU'(x), alpha = 0.1:  e = exp(min(x,0)/alpha)
__device__ __forceinline__ void celu_both(float x, float& h, float& d) {
  const float e = ex2_approx(fminf(x, 0.0f) * (LOG2E / CELU_ALPHA));
  h = x > 0.0f ? x : CELU_ALPHA * (e - 1.0f);
  d = x > 0.0f ? 1.0f : e;
}

// store 16 consecutive K values (columns 16*hf .. 16*hf+15 of a 32-wide chunk) of row r as hi|lo
__device__ __forceinline__ void tc_store_a16(uint8_t* slot, int r, int hf, const float (&v)[16]) {
#pragma unroll
  for (int jj = 0; jj < 4; ++jj) {
    float4 hi, lo;
    tf32_split(v[4 * jj + 0], hi.x, lo.x);
    tf32_split(v[4 * jj + 1], hi.y, lo.y);
    tf32_split(v[4 * jj + 2], hi.z, lo.z);
    tf32_split(v[4 * jj + 3], hi.w, lo.w);
    const uint32_t off = (uint32_t)r * 128u + ((uint32_t)((4 * hf + jj) ^ (r & 7)) << 4);
    *reinterpret_cast<float4*>(slot + off) = hi;
    *reinterpret_cast<float4*>(slot + TC_TM * 128 + off) = lo;
  }
}

template <int N_TERMS>
__global__ void __launch_bounds__(TC_THREADS, 1)
k3_mlp_tc_kernel(const __grid_constant__ TcParams P, const float* __restrict__ aev, float* __restrict__ g,
                 float* __restrict__ e_row) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* base = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* ringA = base;
  uint8_t* ringB = ringA + TC_NA * TC_A_SLOT;
  TcSmem& S = *reinterpret_cast<TcSmem*>(ringB + TC_NB * TC_B_SLOT);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int i = 0; i < TC_NA; ++i) { tc::mbar_init(&S.a_full[i], TC_EPI_THREADS); tc::mbar_init(&S.a_empty[i], 1); }
    for (int i = 0; i < TC_NB; ++i) { tc::mbar_init(&S.b_full[i], 1); tc::mbar_init(&S.b_empty[i], 1); }
    tc::mbar_init(&S.d_full, 1);
    tc::mbar_init(&S.dg_free, TC_EPI_THREADS);
    tc::mbar_fence_init();
  }
  if (warp == 9) tc::tmem_alloc<512>(&S.tmem_base);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tbase = S.tmem_base;

  if (warp < 8) {
    // =========================== producers / epilogue ===========================
    const int q = warp & 3, hf = warp >> 2;
    const int r = 32 * q + lane;                               // tile row == TMEM lane
    const uint32_t tlane = tbase + ((uint32_t)(32 * q) << 16);
    uint32_t ia = 0, nd = 0, ndg = 0;                          // A chunks produced, d_full / dg_free phases seen
    auto acquire = [&]() -> uint8_t* {                         // wait until slot ia%NA is free
      const uint32_t s = ia % TC_NA, use = ia / TC_NA;
      tc::mbar_wait(&S.a_empty[s], (use & 1u) ^ 1u);
      return ringA + s * TC_A_SLOT;
    };
    auto publish = [&]() {
      tc::tc_fence_before();                                   // this thread's tcgen05.ld precede the MMAs that overwrite
      tc::fence_proxy_async_smem();
      tc::mbar_arrive(&S.a_full[ia % TC_NA]);
      ++ia;
    };
    auto wait_d = [&]() { tc::mbar_wait(&S.d_full, nd & 1u); ++nd; tc::tc_fence_after(); };

    for (int tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
      const int row0 = tile * TC_TM;
      int el = 0;
#pragma unroll
      for (int k = 1; k < NSPEC; ++k) el += (row0 >= P.row_start[k]);
      const float* bias = P.bias[el];

      // ---- phase 0 operand: AEV rows, 12 chunks of 32 columns, split into hi|lo ----
      {
        const float4* src = reinterpret_cast<const float4*>(aev + (size_t)row0 * AEV_LEN);
        float4 nxt[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int f = tid + TC_EPI_THREADS * i;
          nxt[i] = __ldg(src + (size_t)(f >> 3) * (AEV_LEN / 4) + (f & 7));
        }
        for (int c = 0; c < D0 / 32; ++c) {
          float4 cur[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) cur[i] = nxt[i];
          if (c + 1 < D0 / 32) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int f = tid + TC_EPI_THREADS * i;
              nxt[i] = __ldg(src + (size_t)(f >> 3) * (AEV_LEN / 4) + 8 * (c + 1) + (f & 7));
            }
          }
          uint8_t* slot = acquire();
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int f = tid + TC_EPI_THREADS * i, rr = f >> 3, j = f & 7;
            float4 hi, lo;
            tf32_split(cur[i].x, hi.x, lo.x); tf32_split(cur[i].y, hi.y, lo.y);
            tf32_split(cur[i].z, hi.z, lo.z); tf32_split(cur[i].w, hi.w, lo.w);
            const uint32_t off = (uint32_t)rr * 128u + ((uint32_t)(j ^ (rr & 7)) << 4);
            *reinterpret_cast<float4*>(slot + off) = hi;
            *reinterpret_cast<float4*>(slot + TC_TM * 128 + off) = lo;
          }
          publish();
        }
      }
      // ---- z1 -> h1 = CELU(z1 + b1): operand of phase 1 ----
      wait_d();
      for (int c = 0; c < D1 / 32; ++c) {
        float z[16], h[16], d;
        tc::tmem_ld16(tlane + 0 + 32 * c + 16 * hf, z);
        const float* b = bias + TC_BIAS_B1 + 32 * c + 16 * hf;
        if (N_TERMS == 3) {
          float sm[16];
          tc::tmem_ld16(tlane + TC_S0_COL + 32 * c + 16 * hf, sm);
          tc::tmem_ld_wait();
#pragma unroll
          for (int k = 0; k < 16; ++k) { const float t = z[k] + sm[k]; z[k] = fmaf(t, P.comp[0], t) + __ldg(b + k); }
        } else {
          tc::tmem_ld_wait();
#pragma unroll
          for (int k = 0; k < 16; ++k) z[k] += __ldg(b + k);
        }
        tc::tmem_st16(tlane + 0 + 32 * c + 16 * hf, z);          // z1 + b1, kept for delta1
#pragma unroll
        for (int k = 0; k < 16; ++k) celu_both(z[k], h[k], d);
        tc::tmem_st_wait();
        uint8_t* slot = acquire();
        tc_store_a16(slot, r, hf, h);
        publish();
      }
      // ---- z2 -> h2: operand of phase 2 ----
      wait_d();
      for (int c = 0; c < D2 / 32; ++c) {
        float z[16], h[16], d;
        tc::tmem_ld16(tlane + 160 + 32 * c + 16 * hf, z);
        tc::tmem_ld_wait();
        const float* b = bias + TC_BIAS_B2 + 32 * c + 16 * hf;
#pragma unroll
        for (int k = 0; k < 16; ++k) celu_both(fmaf(z[k], P.comp[1], z[k]) + __ldg(b + k), h[k], d);
        uint8_t* slot = acquire();
        tc_store_a16(slot, r, hf, h);
        publish();
      }
      // ---- z3 -> e_i = w4.h3 + b4 and delta3 = w4 * CELU'(z3 + b3): operand of phase 3 ----
      wait_d();
      {
        float epart = 0.0f;
        for (int c = 0; c < D3 / 32; ++c) {
          float z[16], dl[16];
          tc::tmem_ld16(tlane + 288 + 32 * c + 16 * hf, z);
          if (N_TERMS == 3) {
            float sm[16];
            tc::tmem_ld16(tlane + TC_S2_COL + 32 * c + 16 * hf, sm);
            tc::tmem_ld_wait();
#pragma unroll
            for (int k = 0; k < 16; ++k) z[k] += sm[k];
          } else {
            tc::tmem_ld_wait();
          }
          const float* b = bias + TC_BIAS_B3 + 32 * c + 16 * hf;
          const float* w4 = bias + TC_BIAS_W4 + 32 * c + 16 * hf;
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            float h, d;
            const float w = __ldg(w4 + k);
            celu_both(fmaf(z[k], P.comp[2], z[k]) + __ldg(b + k), h, d);
            epart = fmaf(w, h, epart);
            dl[k] = w * d;
          }
          uint8_t* slot = acquire();
          tc_store_a16(slot, r, hf, dl);
          publish();
        }
        S.epart[hf][r] = epart;
        asm volatile("bar.sync 1, %0;" ::"n"(TC_EPI_THREADS) : "memory");
        if (hf == 0) e_row[row0 + r] = (S.epart[0][r] + S.epart[1][r]) + __ldg(bias + TC_BIAS_B4);
      }
      // ---- delta2 = d2pre * CELU'(z2 + b2): operand of phase 4 ----
      wait_d();
      for (int c = 0; c < D2 / 32; ++c) {
        float z[16], p[16];
        tc::tmem_ld16(tlane + 160 + 32 * c + 16 * hf, z);
        tc::tmem_ld16(tlane + 384 + 32 * c + 16 * hf, p);
        tc::tmem_ld_wait();
        const float* b = bias + TC_BIAS_B2 + 32 * c + 16 * hf;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          float h, d;
          celu_both(fmaf(z[k], P.comp[1], z[k]) + __ldg(b + k), h, d);
          p[k] = fmaf(p[k], P.comp[3], p[k]) * d;
        }
        uint8_t* slot = acquire();
        tc_store_a16(slot, r, hf, p);
        publish();
      }
      // ---- delta1 = d1pre * CELU'(z1 + b1): operand of the three g passes; drain g ----
      wait_d();
      for (int pass = 0; pass < D0 / TC_GN; ++pass) {
        for (int c = 0; c < D1 / 32; ++c) {
          float z[16], p[16];
          tc::tmem_ld16(tlane + 0 + 32 * c + 16 * hf, z);
          tc::tmem_ld16(tlane + 160 + 32 * c + 16 * hf, p);
          tc::tmem_ld_wait();
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            float h, d;
            celu_both(z[k], h, d);                             // z1 already holds the bias
            p[k] = fmaf(p[k], P.comp[4], p[k]) * d;
          }
          uint8_t* slot = acquire();
          tc_store_a16(slot, r, hf, p);
          publish();
        }
        wait_d();
        float* dst = g + (size_t)(row0 + r) * AEV_LEN + pass * TC_GN + 16 * hf;
#pragma unroll
        for (int c = 0; c < TC_GN / 32; c += 2) {
          float v0[16], v1[16];
          tc::tmem_ld16(tlane + 384 + 32 * c + 16 * hf, v0);
          tc::tmem_ld16(tlane + 384 + 32 * (c + 1) + 16 * hf, v1);
          tc::tmem_ld_wait();
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const float cg = P.comp[5];
            reinterpret_cast<float4*>(dst + 32 * c)[k] =
                make_float4(fmaf(cg, v0[4 * k], v0[4 * k]), fmaf(cg, v0[4 * k + 1], v0[4 * k + 1]),
                            fmaf(cg, v0[4 * k + 2], v0[4 * k + 2]), fmaf(cg, v0[4 * k + 3], v0[4 * k + 3]));
            reinterpret_cast<float4*>(dst + 32 * (c + 1))[k] =
                make_float4(fmaf(cg, v1[4 * k], v1[4 * k]), fmaf(cg, v1[4 * k + 1], v1[4 * k + 1]),
                            fmaf(cg, v1[4 * k + 2], v1[4 * k + 2]), fmaf(cg, v1[4 * k + 3], v1[4 * k + 3]));
          }
        }
        tc::tc_fence_before();
        tc::mbar_arrive(&S.dg_free);
        ++ndg;
      }
    }
  } else if (warp == 8) {
    // =========================== TMA: weight chunks ===========================
    if (lane == 0) {
      uint32_t ib = 0;
      for (int tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        const int row0 = tile * TC_TM;
        int el = 0;
#pragma unroll
        for (int k = 1; k < NSPEC; ++k) el += (row0 >= P.row_start[k]);
        const uint8_t* src = P.wpack + (size_t)el * TC_W_BYTES_PER_ELEM;
#pragma unroll 1
        for (int p = 0; p < TC_NPHASE; ++p) {
          const uint32_t bytes = (uint32_t)tc_chunk_bytes(p);
          const int nk = tc_phase_nk(p);
          for (int c = 0; c < nk; ++c) {
            const uint32_t s = ib % TC_NB, use = ib / TC_NB;
            tc::mbar_wait(&S.b_empty[s], (use & 1u) ^ 1u);
            tc::mbar_arrive_expect_tx(&S.b_full[s], bytes);
            tc::bulk_g2s(ringB + s * TC_B_SLOT, src, bytes, &S.b_full[s]);
            src += bytes;
            ++ib;
          }
        }
      }
    }
  } else {
    // =========================== MMA issuer ===========================
    if (lane == 0) {
      uint32_t ia = 0, ib = 0, ndg = 0;
      for (int tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
#pragma unroll 1
        for (int p = 0; p < TC_NPHASE; ++p) {
          const int N = tc_phase_n(p), nk = tc_phase_nk(p);
          const uint32_t dcol = tbase + (uint32_t)tc_phase_dcol(p);
          const uint32_t idesc = tc::idesc_tf32(TC_TM, N);
          const bool split_acc = N_TERMS == 3 && (p == 0 || p == 2);
          const uint32_t scol = tbase + (uint32_t)(p == 0 ? TC_S0_COL : TC_S2_COL);
          if (p == 3 || p == 4) {
            // p4: d1pre overwrites z2 / z3 / d2pre: every delta2 chunk must exist first (the last
            // chunk's barrier completes after the earlier ones: producers arrive in order);
            // p3: d2pre overwrites S2, which the delta3 producers still read
            const uint32_t il = ia + (uint32_t)nk - 1;
            tc::mbar_wait(&S.a_full[il % TC_NA], (il / TC_NA) & 1u);
          }
          if (p >= 6) {                                   // g pass buffer drained by the epilogue
            tc::mbar_wait(&S.dg_free, ndg & 1u);
            ++ndg;
          }
          for (int c = 0; c < nk; ++c) {
            const uint32_t sa = ia % TC_NA, sb = ib % TC_NB;
            tc::mbar_wait(&S.a_full[sa], (ia / TC_NA) & 1u);
            tc::mbar_wait(&S.b_full[sb], (ib / TC_NB) & 1u);
            tc::tc_fence_after();
            const uint32_t a_hi = tc::smem_u32(ringA + sa * TC_A_SLOT), a_lo = a_hi + TC_TM * 128;
            const uint32_t b_hi = tc::smem_u32(ringB + sb * TC_B_SLOT), b_lo = b_hi + (uint32_t)N * 128;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              const uint64_t dah = tc::smem_desc_sw128(a_hi + 32 * ks), dal = tc::smem_desc_sw128(a_lo + 32 * ks);
              const uint64_t dbh = tc::smem_desc_sw128(b_hi + 32 * ks), dbl = tc::smem_desc_sw128(b_lo + 32 * ks);
              if (split_acc) {
                tc::mma_tf32_ss(scol, dal, dbh, idesc, (c | ks) ? 1u : 0u);
                tc::mma_tf32_ss(scol, dah, dbl, idesc, 1u);
                tc::mma_tf32_ss(dcol, dah, dbh, idesc, (c | ks) ? 1u : 0u);
              } else if (N_TERMS == 3) {
                tc::mma_tf32_ss(dcol, dal, dbh, idesc, (c | ks) ? 1u : 0u);
                tc::mma_tf32_ss(dcol, dah, dbl, idesc, 1u);
                tc::mma_tf32_ss(dcol, dah, dbh, idesc, 1u);
              } else {
                tc::mma_tf32_ss(dcol, dah, dbh, idesc, (c | ks) ? 1u : 0u);
              }
            }
            tc::mma_commit(&S.a_empty[sa]);
            tc::mma_commit(&S.b_empty[sb]);
            ++ia; ++ib;
          }
          tc::mma_commit(&S.d_full);
        }
        ++ndg;                                            // the last pass's drain: consumed below
        tc::mbar_wait(&S.dg_free, (ndg - 1) & 1u);        // keep dg_free phases aligned per tile
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 9) tc::tmem_dealloc<512>(tbase);
}

}  // namespace pfc
