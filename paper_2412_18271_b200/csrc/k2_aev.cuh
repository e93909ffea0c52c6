// k2_aev.cuh -- K2: ANI-style atomic environment vector, forward (O3, O4).
//
// One warp per centre atom.  The radial row is walked 32 entries at a time
// (lane <-> entry): distance, cosine cutoff (SFU cos), and the angular subset
// (d2 < RC2_A, the K1 predicate) is compacted in row order into a per-warp
// shared-memory table of unit vectors.
//   radial  : lane <-> (entry parity, shell k); 4 per-species accumulators,
//             halves combined with one shuffle               (SFU ex2)
//   angular : phase 1, lane <-> triple (j<k): 8 angular factors A_b and 4
//             radial factors W_a = 2 B_a fc_j fc_k into shared memory;
//             phase 2, lane <-> (a,b): out[p][a][b] += A_b W_a in triple
//             order.  No atomics: every accumulator has one owner lane and a
//             fixed summation order, so results are bit-reproducible.
// theta is never formed: cos(theta - theta_b) = c cos(theta_b) + sqrt(1-c^2) sin(theta_b)
// with c = 0.95 cos(phi); the power 32 is five squarings.
// Rows are written in element-sorted padded order (row_of_atom) so K3's tiles
// are contiguous.
#pragma once
#include "pfc_common.cuh"

namespace pfc {

constexpr int AEV_WARPS = 4;

struct AevFwdSmem {
  float4 ur[MAX_ANG];        // unit vector i->j, r
  float2 fs[MAX_ANG];        // fc(r; RC_A), species bits
  float out[AEV_LEN];
  float tA[32][NSHF_Z];
  float tW[32][NSHF_A];
  int tp[32];
  float rr[32], rfc[32];
  int rsp[32];
};

// triple index t in [0, m(m-1)/2) -> (j,k), j<k, lexicographic
__device__ __forceinline__ int tri_row_start(int j, int m) { return (j * (2 * m - j - 1)) >> 1; }
__device__ __forceinline__ void tri_decode(int t, int m, int& j, int& k) {
  float b = (float)(2 * m - 1);
  int jj = (int)((b - sqrtf(b * b - 8.0f * (float)t)) * 0.5f);
  jj = max(0, min(jj, m - 2));
  while (jj < m - 2 && tri_row_start(jj + 1, m) <= t) ++jj;
  while (jj > 0 && tri_row_start(jj, m) > t) --jj;
  j = jj;
  k = jj + 1 + (t - tri_row_start(jj, m));
}

__global__ void __launch_bounds__(AEV_WARPS * 32)
k2_aev_fwd_kernel(int n_atoms, const float4* __restrict__ xs, const float4* __restrict__ xsl,
                  const int* __restrict__ r_off,
                  const int* __restrict__ r_idx, int cap_r, const int* __restrict__ row_of_atom,
                  float* __restrict__ aev, uint32_t* __restrict__ status) {
  __shared__ AevFwdSmem sm[AEV_WARPS];
  const int warp = threadIdx.x >> 5;
  const int i = blockIdx.x * AEV_WARPS + warp;
  if (i >= n_atoms) return;                       // warp-uniform; only __syncwarp below
  AevFwdSmem& S = sm[warp];
  const uint32_t lane = lane_id(), lt = lanemask_lt();
  for (int c = lane; c < AEV_LEN; c += 32) S.out[c] = 0.0f;
  const float4 xi = xs[i], li = xsl[i];
  const int rb = r_off[i];
  const int re = r_off[i + 1] <= cap_r ? r_off[i + 1] : rb;   // capacity overflow (flagged by K1): row unwritten
  int m = 0;
  float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, acc3 = 0.f;
  const int half = lane >> 4;
  const float shf = c_tab.shf_r[lane & 15];
  for (int c0 = rb; c0 < re; c0 += 32) {
    const int e = c0 + (int)lane;
    float r = 1.0f, fcr = 0.0f, dx = 0.f, dy = 0.f, dz = 0.f;
    int sp = 0;
    bool isang = false;
    if (e < re) {
      const int j = r_idx[e];
      const float4 xj = xs[j];
      dx = __fsub_rn(xj.x, xi.x); dy = __fsub_rn(xj.y, xi.y); dz = __fsub_rn(xj.z, xi.z);
      // identical value to K1's predicate (squares do not see the sign)
      const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
      // geometry from the two-float positions (zero low words outside pfc_step)
      const float4 lj = xsl[j];
      dx += lj.x - li.x; dy += lj.y - li.y; dz += lj.z - li.z;
      r = sqrtf(fmaf(dx, dx, fmaf(dy, dy, dz * dz)));
      fcr = 0.5f * __cosf((PI_F / RC_R) * r) + 0.5f;
      sp = __float_as_int(xj.w);
      isang = d2 < RC2_A;
    }
    S.rr[lane] = r; S.rfc[lane] = fcr; S.rsp[lane] = sp;
    const uint32_t mask = __ballot_sync(0xffffffffu, isang);
    if (isang) {
      const int slot = m + __popc(mask & lt);
      if (slot < MAX_ANG) {
        const float rinv = 1.0f / r;
        S.ur[slot] = make_float4(dx * rinv, dy * rinv, dz * rinv, r);
        S.fs[slot] = make_float2(0.5f * __cosf((PI_F / RC_A) * r) + 0.5f, __int_as_float(sp));
      }
    }
    m += __popc(mask);
    __syncwarp();
    const int nin = min(32, re - c0);
    for (int n = half; n < nin; n += 2) {
      const float dr = S.rr[n] - shf;
      const float v = 0.25f * ex2_approx(-(ETA_R * LOG2E) * dr * dr) * S.rfc[n];
      const int s = S.rsp[n];
      acc0 += (s == 0) ? v : 0.0f;
      acc1 += (s == 1) ? v : 0.0f;
      acc2 += (s == 2) ? v : 0.0f;
      acc3 += (s == 3) ? v : 0.0f;
    }
    __syncwarp();
  }
  acc0 += __shfl_xor_sync(0xffffffffu, acc0, 16);
  acc1 += __shfl_xor_sync(0xffffffffu, acc1, 16);
  acc2 += __shfl_xor_sync(0xffffffffu, acc2, 16);
  acc3 += __shfl_xor_sync(0xffffffffu, acc3, 16);
  if (lane < 16) {
    S.out[lane] = acc0; S.out[16 + lane] = acc1; S.out[32 + lane] = acc2; S.out[48 + lane] = acc3;
  }
  if (m > MAX_ANG) {
    if (lane == 0) atomicOr(status, ST_ANGULAR_ROW);
    m = MAX_ANG;
  }
  __syncwarp();
  // ---- angular ----
  const int T = (m * (m - 1)) >> 1;
  const int pa = lane >> 3, pb = lane & 7;
  for (int t0 = 0; t0 < T; t0 += 32) {
    const int t = t0 + (int)lane;
    if (t < T) {
      int j, k;
      tri_decode(t, m, j, k);
      const float4 uj = S.ur[j], uk = S.ur[k];
      const float2 fj = S.fs[j], fk = S.fs[k];
      const float c = COS_SCALE * (uj.x * uk.x + uj.y * uk.y + uj.z * uk.z);
      const float s = sqrtf(fmaf(-c, c, 1.0f));
      const float rbar = 0.5f * (uj.w + uk.w);
      const float w2 = 2.0f * fj.x * fk.x;
#pragma unroll
      for (int b = 0; b < NSHF_Z; ++b) {
        float q = fmaf(0.5f, fmaf(c, c_tab.cos_z[b], s * c_tab.sin_z[b]), 0.5f);
        q *= q; q *= q; q *= q; q *= q; q *= q;                   // ^32
        S.tA[lane][b] = q;
      }
#pragma unroll
      for (int a = 0; a < NSHF_A; ++a) {
        const float dr = rbar - c_tab.shf_a[a];
        S.tW[lane][a] = w2 * ex2_approx(-(ETA_A * LOG2E) * dr * dr);
      }
      S.tp[lane] = pair_block(__float_as_int(fj.y), __float_as_int(fk.y));
    }
    __syncwarp();
    const int nt = min(32, T - t0);
    int pcur = S.tp[0];
    float acc = 0.0f;
    for (int n = 0; n < nt; ++n) {
      const int p = S.tp[n];
      if (p != pcur) {                                            // warp-uniform
        S.out[RAD_LEN + 32 * pcur + lane] += acc;
        acc = 0.0f; pcur = p;
      }
      acc = fmaf(S.tA[n][pb], S.tW[n][pa], acc);
    }
    S.out[RAD_LEN + 32 * pcur + lane] += acc;
    __syncwarp();
  }
  float* dst = aev + (size_t)row_of_atom[i] * AEV_LEN;
  for (int c = lane; c < AEV_LEN; c += 32) dst[c] = S.out[c];
}

}  // namespace pfc
