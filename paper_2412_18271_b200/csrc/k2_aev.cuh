// k2_aev.cuh -- K2: ANI-style atomic environment vector, forward (O3, O4).
//
// One warp per centre atom.  The neighbour row (K1's entry words: index, species, angular flag)
// is walked 32 entries at a time (lane <-> entry): distance and unit vector (one MUFU.RSQ +
// Newton), cosine cutoff (SFU cos); the chunk is staged in shared memory GROUPED BY SPECIES (four
// ballots), and the angular subset is compacted in row order into a per-warp table of unit
// vectors plus one slot list per species.
//   radial  : lane <-> (entry parity, shell k); one loop per species segment, so each of the four
//             accumulators is a plain sum  (SFU ex2)
//   angular : the triples are enumerated BLOCK BY BLOCK of the species-pair index p
//             (HH HC HN HO CC CN CO NN NO OO): block (s1,s2) holds the pairs of list s1 x list s2
//             (s1 < s2) or the unordered pairs of list s1 in round-robin (circulant) order -- an
//             order that decodes without a square root or a search loop.  Every block is padded to a
//             multiple of four slots (padding slots contribute exact zeros).
//             phase 1, lane <-> slot: the 8 angular factors A_b and the 4 radial factors
//             W_a = 2 B_a fc_j fc_k of the triple, written TRANSPOSED into shared memory
//             (tA[b][slot], tW[a][slot]: conflict-free stores);
//             phase 2, lane <-> output (a, b): one register accumulator per block p; a block's slots
//             are read four at a time (one LDS.128 per operand, four FMAs): 1.5 instructions per
//             triple where the earlier slot-major layout cost 3 and a shared-memory flush per block
//             and chunk.  The ten accumulators go straight to global memory.
//             No atomics: every accumulator has one owner lane and a fixed summation order, so
//             results are bit-reproducible.
// theta is never formed: cos(theta - theta_b) = c cos(theta_b) + sqrt(1-c^2) sin(theta_b)
// with c = 0.95 cos(phi); the power 32 is five squarings.
// Rows are written in element-sorted padded order (row_of_atom) so K3's tiles are contiguous --
// as fp32 rows aev[row][384] for the FP32 MLP, or (PACK16) directly as the A operand image of the
// tensor-core MLP's first GEMM: per 128-row tile and 32-column chunk one 16 KB block, the values
// times 8 split into fp16 hi | lo, K-major SWIZZLE_64B (k3_mlp_tc.cuh) -- the AEV -> MLP fusion of
// SURVEY.md 8(f) item 4 on the operand side: K3 brings a chunk in with one bulk copy and no warp
// touches it again.
#pragma once
#include <cuda_fp16.h>

#include "aev_common.cuh"

namespace pfc {

#ifndef PFC_K2_TCH
#define PFC_K2_TCH 96
#endif
#ifndef PFC_K2_MINB
#define PFC_K2_MINB 24
#endif
constexpr int K2_TCH = PFC_K2_TCH;               // padded triple slots per chunk (3 passes of 32 lanes)
constexpr int K2_TLD = K2_TCH + 4;               // row stride of the transposed factor tables: 4 mod 32 banks

struct AevFwdSmem {
  float4 ur[MAX_ANG];            // unit vector i->j, r         (row order)
  float fc[MAX_ANG];             // fc(r; RC_A)
  uint8_t lst[NSPEC][MAX_ANG];   // table slots of each species, ascending
  float tA[NSHF_Z][K2_TLD];      // A_b of the staged slots, transposed
  float tW[NSHF_A][K2_TLD];      // W_a of the staged slots, transposed
  float2 rad[32];                // (r, fc(r; RC_R)) of one radial chunk, grouped by species
  int pre4[NPAIR + 1];           // first 4-slot group of each species-pair block
};

constexpr int K2_PACK_CHUNK_BYTES = 2 * 128 * 64;     // == TC_A_SLOT: hi block then lo block of one [128 x 32] chunk
constexpr float K2_PACK_SCALE = 8.0f;                // == 2^TC_AEV_SCALE_LOG2

template <bool PACK16>
__global__ void __launch_bounds__(AEV_WARPS * 32, PFC_K2_MINB)
k2_aev_fwd_kernel(int n_atoms, const float4* __restrict__ xs, const float4* __restrict__ xsl,
                  const int* __restrict__ row_beg, const uint32_t* __restrict__ nbr, const int2* __restrict__ cnt,
                  const int* __restrict__ row_of_atom,
                  float* __restrict__ aev, uint32_t* __restrict__ status) {
  __shared__ __align__(16) AevFwdSmem sm[AEV_WARPS];
  const int warp = threadIdx.x >> 5;
  const int i = blockIdx.x * AEV_WARPS + warp;
  if (i >= n_atoms) return;                       // warp-uniform; only __syncwarp below
  AevFwdSmem& S = sm[warp];
  const uint32_t lane = lane_id(), lt = lanemask_lt();
  const float4 xi = xs[i], li = xsl[i];
  const int rb = row_beg[i];
  const int re = rb + cnt[i].x;
  const int row = row_of_atom[i];
  float* dst = aev + (size_t)row * AEV_LEN;
  // one 32-column chunk of my row: lane <-> column.  PACK16: my fp16 element of the chunk image (the 32
  // lanes fill one 64-byte row of the hi block and one of the lo block)
  uint8_t* pk = nullptr;
  if (PACK16) {
    const uint32_t r = (uint32_t)row & 127u, k = lane;
    pk = reinterpret_cast<uint8_t*>(aev) + (size_t)(row >> 7) * (AEV_LEN / 32) * K2_PACK_CHUNK_BYTES +
         (r >> 3) * 512u + (r & 7u) * 64u + ((((k >> 3) ^ ((r >> 1) & 3u)) << 4) | ((k & 7u) << 1));
  }
  auto emit = [&](int c, float v) {
    if (!PACK16) {
      dst[32 * c + (int)lane] = v;
    } else {
      const float sv = K2_PACK_SCALE * v;
      const __half h = __float2half_rn(sv);
      const __half l = __float2half_rn(sv - __half2float(h));
      *reinterpret_cast<__half*>(pk + (size_t)c * K2_PACK_CHUNK_BYTES) = h;
      *reinterpret_cast<__half*>(pk + (size_t)c * K2_PACK_CHUNK_BYTES + K2_PACK_CHUNK_BYTES / 2) = l;
    }
  };
  int m = 0;
  uint32_t na = 0;                                // angular neighbours per species, one byte each
  float acc[NSPEC] = {0.f, 0.f, 0.f, 0.f};
  const int half = lane >> 4;
  const float shf = c_tab.shf_r[lane & 15];
  for (int c0 = rb; c0 < re; c0 += 32) {
    const int e = c0 + (int)lane;
    NbrGeom g;
    g.sp = -1; g.ang = false; g.r = 1.0f; g.ux = g.uy = g.uz = 0.0f;
    float fcr = 0.0f;
    if (e < re) {
      g = nbr_geometry(nbr[e], xi, li, xs, xsl);
      fcr = 0.5f * __cosf((PI_F / RC_R) * g.r) + 0.5f;
    }
    // stage (r, fc) grouped by species; angular entries go to the table (row order) and to
    // the slot list of their species
    int seg[NSPEC + 1];
    seg[0] = 0;
    int pos = 0, lpos = 0;
    const uint32_t amask = __ballot_sync(0xffffffffu, g.ang);
#pragma unroll
    for (int z = 0; z < NSPEC; ++z) {
      const uint32_t mz = __ballot_sync(0xffffffffu, g.sp == z);
      const uint32_t az = mz & amask;
      if (g.sp == z) {
        pos = seg[z] + __popc(mz & lt);
        lpos = (int)((na >> (8 * z)) & 255u) + __popc(az & lt);
      }
      seg[z + 1] = seg[z] + __popc(mz);
      na += (uint32_t)__popc(az) << (8 * z);      // (a count above 96 is flagged below; bytes cannot carry: m <= 128)
    }
    if (g.sp >= 0) S.rad[pos] = make_float2(g.r, fcr);
    if (g.ang) {
      const int slot = m + __popc(amask & lt);
      if (slot < MAX_ANG) {
        S.ur[slot] = make_float4(g.ux, g.uy, g.uz, g.r);
        S.fc[slot] = 0.5f * __cosf((PI_F / RC_A) * g.r) + 0.5f;
        S.lst[g.sp][lpos] = (uint8_t)slot;        // lpos <= slot < MAX_ANG
      }
    }
    m += __popc(amask);
    __syncwarp();
#pragma unroll
    for (int z = 0; z < NSPEC; ++z) {
      for (int n = seg[z] + half; n < seg[z + 1]; n += 2) {
        const float2 v = S.rad[n];
        const float dr = v.x - shf;
        acc[z] = fmaf(ex2_approx(-(ETA_R * LOG2E) * dr * dr), v.y, acc[z]);
      }
    }
    __syncwarp();
  }
  // radial part of the row: lanes 0-15 hold shell k of species 0 / 2, lanes 16-31 of species 1 / 3
#pragma unroll
  for (int z = 0; z < NSPEC; ++z) acc[z] += __shfl_xor_sync(0xffffffffu, acc[z], 16);
  emit(0, 0.25f * (half ? acc[1] : acc[0]));
  emit(1, 0.25f * (half ? acc[3] : acc[2]));
  if (m > MAX_ANG) {                              // outputs unspecified (S25); keep every index in range
    if (lane == 0) atomicOr(status, ST_ANGULAR_ROW);
    m = 0; na = 0;
  }
  // ---- angular ----
  // block sizes -> prefix table in units of four slots (every lane computes the same ten numbers)
  const int nH = (int)(na & 255u), nC = (int)((na >> 8) & 255u), nN = (int)((na >> 16) & 255u), nO = (int)(na >> 24);
  int pre4[NPAIR + 1];
  {
    const int sz[NPAIR] = {(nH * (nH - 1)) >> 1, nH * nC, nH * nN, nH * nO, (nC * (nC - 1)) >> 1,
                           nC * nN, nC * nO, (nN * (nN - 1)) >> 1, nN * nO, (nO * (nO - 1)) >> 1};
    pre4[0] = 0;
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) pre4[p + 1] = pre4[p] + ((sz[p] + 3) >> 2);
  }
  if (lane == 0) {
#pragma unroll
    for (int p = 0; p <= NPAIR; ++p) S.pre4[p] = pre4[p];
  }
  __syncwarp();
  const int n_slots = 4 * pre4[NPAIR];
  const int pa = lane >> 3, pb = lane & 7;        // phase 2: my output (a, b)
  float out[NPAIR];
#pragma unroll
  for (int p = 0; p < NPAIR; ++p) out[p] = 0.0f;
  for (int s0 = 0; s0 < n_slots; s0 += K2_TCH) {
#pragma unroll
    for (int pass = 0; pass < K2_TCH / 32; ++pass) {
      const int s = s0 + 32 * pass + (int)lane;
      if (s0 + 32 * pass >= n_slots) break;       // warp-uniform
      float2 A2[NSHF_Z / 2];
      float2 W2[NSHF_A / 2];
#pragma unroll
      for (int b = 0; b < NSHF_Z / 2; ++b) A2[b] = make_float2(0.f, 0.f);
      W2[0] = W2[1] = make_float2(0.f, 0.f);
      if (s < n_slots) {
        // block of my slot: branch-free count over the ten (warp-uniform) block starts
        int p = 0;
#pragma unroll
        for (int k = 1; k < NPAIR; ++k) p += ((s >> 2) >= pre4[k]) ? 1 : 0;
        const int q = s - 4 * S.pre4[p];
        const int s1 = (int)((0xE9500u >> (2 * p)) & 3u), s2 = (int)((0xFB9E4u >> (2 * p)) & 3u);   // 0000111223 / 0123123233
        const int n1 = (int)((na >> (8 * s1)) & 255u), n2 = (int)((na >> (8 * s2)) & 255u);
        int jj, kk;
        bool valid;
        if (s1 == s2) {
          // unordered pairs of n1 items in round-robin order: q = (d - 1) n1 + a  ->  {a, (a + d) mod n1}
          const int d1 = small_div(q, n1);
          jj = q - d1 * n1;
          kk = jj + d1 + 1;
          kk = kk >= n1 ? kk - n1 : kk;
          valid = q < ((n1 * (n1 - 1)) >> 1);
        } else {
          jj = small_div(q, n2);
          kk = q - jj * n2;
          valid = q < n1 * n2;
        }
        if (valid) {
          const int j = S.lst[s1][jj], k = S.lst[s2][kk];
          const float4 uj = S.ur[j], uk = S.ur[k];
          const float c = COS_SCALE * (uj.x * uk.x + uj.y * uk.y + uj.z * uk.z);
          const float sn = sqrt_newton(fmaf(-c, c, 1.0f));
          const float rbar = 0.5f * (uj.w + uk.w);
          const float w2 = 2.0f * S.fc[j] * S.fc[k];
          const float2 cc2 = make_float2(c, c), ss2 = make_float2(sn, sn), half2 = make_float2(0.5f, 0.5f);
#pragma unroll
          for (int b = 0; b < NSHF_Z / 2; ++b) {                      // two shifts at a time (packed fp32 pairs)
            const float2 cz = make_float2(0.5f * c_tab.cos_z[2 * b], 0.5f * c_tab.cos_z[2 * b + 1]);
            const float2 sz = make_float2(0.5f * c_tab.sin_z[2 * b], 0.5f * c_tab.sin_z[2 * b + 1]);
            float2 q1 = pk_fma(cc2, cz, pk_fma(ss2, sz, half2));      // (1 + cos(theta - theta_b)) / 2
            q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1);   // ^32
            A2[b] = q1;
          }
          const float2 rb2 = make_float2(rbar, rbar), m1 = make_float2(-1.0f, -1.0f), ww2 = make_float2(w2, w2),
                       ke = make_float2(-(ETA_A * LOG2E), -(ETA_A * LOG2E));
#pragma unroll
          for (int a = 0; a < NSHF_A / 2; ++a) {
            const float2 dr = pk_fma(make_float2(c_tab.shf_a[2 * a], c_tab.shf_a[2 * a + 1]), m1, rb2);
            const float2 arg = pk_mul(pk_mul(dr, dr), ke);
            W2[a] = pk_mul(ww2, make_float2(ex2_approx(arg.x), ex2_approx(arg.y)));
          }
        }
      }
      const int col = 32 * pass + (int)lane;
#pragma unroll
      for (int b = 0; b < NSHF_Z / 2; ++b) { S.tA[2 * b][col] = A2[b].x; S.tA[2 * b + 1][col] = A2[b].y; }
      S.tW[0][col] = W2[0].x; S.tW[1][col] = W2[0].y; S.tW[2][col] = W2[1].x; S.tW[3][col] = W2[1].y;
    }
    __syncwarp();
    // phase 2: the groups of four slots of every block that fall into this chunk
    const int g0 = s0 >> 2, g1 = min(n_slots, s0 + K2_TCH) >> 2;
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
      const int lo = max(pre4[p], g0), hi = min(pre4[p + 1], g1);
      float a0 = out[p], a1 = 0.0f;
#pragma unroll 1
      for (int g = lo; g < hi; ++g) {
        const float4 A = *reinterpret_cast<const float4*>(&S.tA[pb][4 * (g - g0)]);
        const float4 W = *reinterpret_cast<const float4*>(&S.tW[pa][4 * (g - g0)]);
        a0 = fmaf(A.x, W.x, a0); a1 = fmaf(A.y, W.y, a1);
        a0 = fmaf(A.z, W.z, a0); a1 = fmaf(A.w, W.w, a1);
      }
      out[p] = a0 + a1;
    }
    __syncwarp();
  }
#pragma unroll
  for (int p = 0; p < NPAIR; ++p) emit(2 + p, out[p]);
}

// pfc_get_intermediates on the tensor path: the packed operand image back to fp32 rows
// (aev = (hi + lo) / 8: the value the tensor core multiplies, within 2^-23 of K2's fp32 sum)
__global__ void k2_unpack16_kernel(int n_rows, const uint8_t* __restrict__ packed, float* __restrict__ aev) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_rows * AEV_LEN) return;
  const uint32_t row = (uint32_t)(idx / AEV_LEN), col = (uint32_t)(idx % AEV_LEN), r = row & 127u, k = col & 31u;
  const uint8_t* blk = packed + ((size_t)(row >> 7) * (AEV_LEN / 32) + (size_t)(col >> 5)) * K2_PACK_CHUNK_BYTES +
                       (r >> 3) * 512u + (r & 7u) * 64u + ((((k >> 3) ^ ((r >> 1) & 3u)) << 4) | ((k & 7u) << 1));
  const float hi = __half2float(*reinterpret_cast<const __half*>(blk));
  const float lo = __half2float(*reinterpret_cast<const __half*>(blk + K2_PACK_CHUNK_BYTES / 2));
  aev[idx] = (hi + lo) * (1.0f / K2_PACK_SCALE);
}

}  // namespace pfc
