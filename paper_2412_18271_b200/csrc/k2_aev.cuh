// k2_aev.cuh -- K2: ANI-style atomic environment vector, forward (O3, O4).
//
// One warp per centre atom.  The radial row is walked 32 entries at a time
// (lane <-> entry): distance, cosine cutoff (SFU cos); the chunk is staged in
// shared memory GROUPED BY SPECIES (four ballots), and the angular subset
// (d2 < RC2_A, the K1 predicate) is compacted in row order into a per-warp
// table of unit vectors plus one index list per species.
//   radial  : lane <-> (entry parity, shell k); one loop per species segment, so
//             each of the four accumulators is a plain sum  (SFU ex2)
//   angular : triples are enumerated BLOCK BY BLOCK of the species-pair index p
//             (HH HC HN HO CC CN CO NN NO OO): block (s1,s2) holds the pairs of
//             list s1 x list s2 (s1 < s2) or the unordered pairs of list s1.
//             phase 1, lane <-> triple: 8 angular factors A_b and 4 radial factors
//             W_a = 2 B_a fc_j fc_k into shared memory;
//             phase 2, lane <-> (a,b): out[p][a][b] += A_b W_a over the staged
//             triples of one block at a time -- the block of a staged triple is
//             known from the prefix table, so the inner loop is two loads and an
//             FMA, and an accumulator is flushed once per block and chunk (the
//             per-triple block test of the earlier lexicographic order cost 43 % of
//             the kernel's instructions).
//             No atomics: every accumulator has one owner lane and a fixed
//             summation order, so results are bit-reproducible.
// theta is never formed: cos(theta - theta_b) = c cos(theta_b) + sqrt(1-c^2) sin(theta_b)
// with c = 0.95 cos(phi); the power 32 is five squarings.
// Rows are written in element-sorted padded order (row_of_atom) so K3's tiles
// are contiguous.
#pragma once
#include "pfc_common.cuh"

namespace pfc {

constexpr int AEV_WARPS = 4;

struct AevFwdSmem {
  float4 ur[MAX_ANG];        // unit vector i->j, r         (row order)
  float fc[MAX_ANG];         // fc(r; RC_A)
  uint8_t lst[NSPEC][MAX_ANG];   // table slots of each species, ascending
  float out[AEV_LEN];
  float tA[32][NSHF_Z];
  float tW[32][NSHF_A];
  float2 rad[32];            // (r, fc(r; RC_R)) of one radial chunk, grouped by species
  int pre[NPAIR + 1];        // first triple of each species-pair block
};

// species pair of block p (nibble tables):  s1 = 0000111223, s2 = 0123123233
__device__ __forceinline__ int block_s1(int p) { return (int)((0x3221110000ull >> (4 * p)) & 3ull); }
__device__ __forceinline__ int block_s2(int p) { return (int)((0x3323213210ull >> (4 * p)) & 3ull); }

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
  const float4 xi = xs[i], li = xsl[i];
  const int rb = r_off[i];
  const int re = r_off[i + 1] <= cap_r ? r_off[i + 1] : rb;   // capacity overflow (flagged by K1): row unwritten
  int m = 0;
  uint32_t na = 0;                                // angular neighbours per species, one byte each
  float acc[NSPEC] = {0.f, 0.f, 0.f, 0.f};
  const int half = lane >> 4;
  const float shf = c_tab.shf_r[lane & 15];
  for (int c0 = rb; c0 < re; c0 += 32) {
    const int e = c0 + (int)lane;
    float r = 1.0f, fcr = 0.0f, dx = 0.f, dy = 0.f, dz = 0.f;
    int sp = -1;
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
    // stage (r, fc) grouped by species; angular entries go to the table (row order) and to
    // the index list of their species
    int seg[NSPEC + 1];
    seg[0] = 0;
    int pos = 0, lpos = 0;
    const uint32_t amask = __ballot_sync(0xffffffffu, isang);
#pragma unroll
    for (int z = 0; z < NSPEC; ++z) {
      const uint32_t mz = __ballot_sync(0xffffffffu, sp == z);
      const uint32_t az = mz & amask;
      if (sp == z) {
        pos = seg[z] + __popc(mz & lt);
        lpos = (int)((na >> (8 * z)) & 255u) + __popc(az & lt);
      }
      seg[z + 1] = seg[z] + __popc(mz);
      na += (uint32_t)__popc(az) << (8 * z);      // (a count above 96 is flagged below; bytes cannot carry: m <= 128)
    }
    if (sp >= 0) S.rad[pos] = make_float2(r, fcr);
    if (isang) {
      const int slot = m + __popc(amask & lt);
      if (slot < MAX_ANG) {
        const float rinv = 1.0f / r;
        S.ur[slot] = make_float4(dx * rinv, dy * rinv, dz * rinv, r);
        S.fc[slot] = 0.5f * __cosf((PI_F / RC_A) * r) + 0.5f;
        S.lst[sp][lpos] = (uint8_t)slot;          // lpos <= slot < MAX_ANG
      }
    }
    m += __popc(amask);
    __syncwarp();
#pragma unroll
    for (int z = 0; z < NSPEC; ++z) {
      for (int n = seg[z] + half; n < seg[z + 1]; n += 2) {
        const float2 v = S.rad[n];
        const float dr = v.x - shf;
        acc[z] = fmaf(0.25f * ex2_approx(-(ETA_R * LOG2E) * dr * dr), v.y, acc[z]);
      }
    }
    __syncwarp();
  }
#pragma unroll
  for (int z = 0; z < NSPEC; ++z) {
    acc[z] += __shfl_xor_sync(0xffffffffu, acc[z], 16);
    if (lane < 16) S.out[NSHF_R * z + lane] = acc[z];
  }
  for (int c = RAD_LEN + (int)lane; c < AEV_LEN; c += 32) S.out[c] = 0.0f;
  if (m > MAX_ANG) {                              // outputs unspecified (S25); keep every index in range
    if (lane == 0) atomicOr(status, ST_ANGULAR_ROW);
    m = 0; na = 0;
  }
  // ---- angular ----
  // block sizes -> prefix table (every lane computes the same ten numbers)
  {
    int run = 0;
    if (lane == 0) S.pre[0] = 0;
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
      const int n1 = (int)((na >> (8 * block_s1(p))) & 255u), n2 = (int)((na >> (8 * block_s2(p))) & 255u);
      run += block_s1(p) == block_s2(p) ? (n1 * (n1 - 1)) >> 1 : n1 * n2;
      if (lane == 0) S.pre[p + 1] = run;
    }
  }
  __syncwarp();
  const int T = (m * (m - 1)) >> 1;               // == S.pre[NPAIR]
  const int pa = lane >> 3, pb = lane & 7;
  int bcur = 0;                                   // block of the first staged triple (warp-uniform)
  for (int t0 = 0; t0 < T; t0 += 32) {
    const int t = t0 + (int)lane;
    if (t < T) {
      int p = bcur;
      while (t >= S.pre[p + 1]) ++p;
      const int q = t - S.pre[p];
      const int s1 = block_s1(p), s2 = block_s2(p);
      int jj, kk;
      if (s1 == s2) {
        tri_decode(q, (int)((na >> (8 * s1)) & 255u), jj, kk);
      } else {
        const int n2 = (int)((na >> (8 * s2)) & 255u);
        jj = (int)(((float)q + 0.5f) / (float)n2);      // exact: q < 2^13
        kk = q - jj * n2;
      }
      const int j = S.lst[s1][jj], k = S.lst[s2][kk];
      const float4 uj = S.ur[j], uk = S.ur[k];
      const float c = COS_SCALE * (uj.x * uk.x + uj.y * uk.y + uj.z * uk.z);
      const float s = sqrtf(fmaf(-c, c, 1.0f));
      const float rbar = 0.5f * (uj.w + uk.w);
      const float w2 = 2.0f * S.fc[j] * S.fc[k];
      const float2 cc2 = make_float2(c, c), ss2 = make_float2(s, s), half2 = make_float2(0.5f, 0.5f);
#pragma unroll
      for (int b = 0; b < NSHF_Z / 2; ++b) {                        // two shifts at a time (packed fp32 pairs)
        const float2 cz = make_float2(c_tab.cos_z[2 * b], c_tab.cos_z[2 * b + 1]);
        const float2 sz = make_float2(c_tab.sin_z[2 * b], c_tab.sin_z[2 * b + 1]);
        float2 q1 = pk_fma(half2, pk_fma(cc2, cz, pk_mul(ss2, sz)), half2);
        q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1); q1 = pk_mul(q1, q1);   // ^32
        *reinterpret_cast<float2*>(&S.tA[lane][2 * b]) = q1;
      }
#pragma unroll
      for (int a = 0; a < NSHF_A; ++a) {
        const float dr = rbar - c_tab.shf_a[a];
        S.tW[lane][a] = w2 * ex2_approx(-(ETA_A * LOG2E) * dr * dr);
      }
    }
    __syncwarp();
    const int nt = min(32, T - t0);
    int n = 0;
    while (n < nt) {                               // one pass per block present in this chunk
      while (t0 + n >= S.pre[bcur + 1]) ++bcur;
      const int hi = min(nt, S.pre[bcur + 1] - t0);
      float a2 = 0.0f;
#pragma unroll 4
      for (; n < hi; ++n) a2 = fmaf(S.tA[n][pb], S.tW[n][pa], a2);
      S.out[RAD_LEN + 32 * bcur + lane] += a2;
    }
    __syncwarp();
  }
  float* dst = aev + (size_t)row_of_atom[i] * AEV_LEN;
  for (int c = lane; c < AEV_LEN; c += 32) dst[c] = S.out[c];
}

}  // namespace pfc
