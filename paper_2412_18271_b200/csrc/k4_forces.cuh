// k4_forces.cuh -- K4: chain rule from g_i = dE/dAEV_i to per-atom forces, with
// fixed-order accumulation (O7; "forces by backprop").
//
// K4a (centre-owned, one warp per atom i): recomputes the pair/triple geometry
// and writes, for every radial CSR entry e = (i -> j),
//      edge[e] = P_e = sum_a g_i[a] * dAEV_i[a]/dx_j        (gradient, not force)
// plus self[i] = sum_e P_e.  By translation invariance dE_i/dx_i = -self[i].
//   radial : lane <-> entry, 16 shells.
//   angular: phase 1, lane <-> triple (j<k): the three scalars
//            C = dE/dcos(phi), Rj = dE/dr_j, Rk = dE/dr_k into shared memory;
//            phase 2, lane <-> angular neighbour n sums over its partners k in
//            index order:  grad_n = (sum_k C u_k - (sum_k C cos(phi)) u_n)/r_n
//                                   + (sum_k R) u_n.
// K4b (gather, one warp per atom a):
//      F_a = self[a] - sum_{e in row(a), ascending} edge[rev(e)]
// where rev(a->j) is the position of a in row j (binary search; lists are
// symmetric and sorted).  No float atomics anywhere.
#pragma once
#include "k2_aev.cuh"

namespace pfc {

constexpr int K4_TCH = 128;              // triples per shared-memory pass
constexpr int GA_STRIDE = 36;            // padded stride of one 32-float g block

struct AevBwdSmem {
  float4 ur[MAX_ANG];                    // unit vector, r
  float4 fs[MAX_ANG];                    // fc, dfc (RC_A), species bits, entry index bits
  float4 pr[MAX_ANG];                    // radial part of P for this neighbour
  float gR[RAD_LEN];
  float gA[NPAIR * GA_STRIDE];
  float tC[K4_TCH], tJ[K4_TCH], tK[K4_TCH];
};

__global__ void __launch_bounds__(AEV_WARPS * 32)
k4a_aev_bwd_kernel(int n_atoms, const float4* __restrict__ xs, const float4* __restrict__ xsl,
                   const int* __restrict__ r_off,
                   const int* __restrict__ r_idx, int cap_r, const int* __restrict__ row_of_atom,
                   const float* __restrict__ g, float4* __restrict__ edge, float4* __restrict__ self) {
  __shared__ AevBwdSmem sm[AEV_WARPS];
  const int warp = threadIdx.x >> 5;
  const int i = blockIdx.x * AEV_WARPS + warp;
  if (i >= n_atoms) return;
  AevBwdSmem& S = sm[warp];
  const uint32_t lane = lane_id(), lt = lanemask_lt();
  {
    // g_i: 96 granules of 16 bytes, three per lane, fetched asynchronously -- the HBM latency of
    // this row overlaps the neighbour gathers below (it was 39 % of the kernel's stall samples
    // when loaded synchronously)
    const float* src = g + (size_t)row_of_atom[i] * AEV_LEN;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const int c = 4 * ((int)lane + 32 * q);
      float* dst = c < RAD_LEN ? S.gR + c : S.gA + ((c - RAD_LEN) >> 5) * GA_STRIDE + ((c - RAD_LEN) & 31);
      cp_async16(dst, src + c);
    }
    cp_async_commit();
  }
  bool g_pending = true;
  const float4 xi = xs[i], li = xsl[i];
  const int rb = r_off[i];
  const int re = r_off[i + 1] <= cap_r ? r_off[i + 1] : rb;   // capacity overflow (flagged by K1): row unwritten
  int m = 0;
  float sx = 0.f, sy = 0.f, sz = 0.f;            // this lane's share of self[i]
  for (int c0 = rb; c0 < re; c0 += 32) {
    const int e = c0 + (int)lane;
    bool isang = false;
    float px = 0.f, py = 0.f, pz = 0.f, ux = 0.f, uy = 0.f, uz = 0.f, r = 1.f;
    float fc = 0.f, dfc = 0.f;
    int sp = 0;
    if (e < re) {
      const int j = r_idx[e];
      const float4 xj = xs[j];
      float dx = __fsub_rn(xj.x, xi.x), dy = __fsub_rn(xj.y, xi.y), dz = __fsub_rn(xj.z, xi.z);
      const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
      const float4 lj = xsl[j];                  // same two-float geometry as K2
      dx += lj.x - li.x; dy += lj.y - li.y; dz += lj.z - li.z;
      r = sqrtf(fmaf(dx, dx, fmaf(dy, dy, dz * dz)));
      const float rinv = 1.0f / r;
      ux = dx * rinv; uy = dy * rinv; uz = dz * rinv;
      sp = __float_as_int(xj.w);
      isang = d2 < RC2_A;
      float sn, cs;
      __sincosf((PI_F / RC_R) * r, &sn, &cs);
      fc = 0.5f * cs + 0.5f; dfc = -(PI_F / (2.0f * RC_R)) * sn;
    }
    if (g_pending) {                             // warp-uniform: every lane's granules, then the handover
      cp_async_wait<0>();
      __syncwarp();
      g_pending = false;
    }
    if (e < re) {
      // two shells at a time in packed fp32 pairs (the exponentials stay scalar SFU calls)
      const float2* gs = reinterpret_cast<const float2*>(S.gR + NSHF_R * sp);
      const float2 r2 = make_float2(r, r), m1 = make_float2(-1.0f, -1.0f), fc2 = make_float2(fc, fc),
                   dfc2 = make_float2(dfc, dfc), ke = make_float2(-(ETA_R * LOG2E), -(ETA_R * LOG2E)),
                   k2e = make_float2(-2.0f * ETA_R, -2.0f * ETA_R);
      float2 d2acc = make_float2(0.0f, 0.0f);
#pragma unroll
      for (int k = 0; k < NSHF_R / 2; ++k) {
        const float2 dr = pk_fma(make_float2(c_tab.shf_r[2 * k], c_tab.shf_r[2 * k + 1]), m1, r2);
        const float2 arg = pk_mul(pk_mul(dr, dr), ke);
        const float2 ex = make_float2(ex2_approx(arg.x), ex2_approx(arg.y));
        d2acc = pk_fma(pk_mul(gs[k], ex), pk_fma(pk_mul(dr, k2e), fc2, dfc2), d2acc);
      }
      float dEdr = 0.25f * (d2acc.x + d2acc.y);
      px = dEdr * ux; py = dEdr * uy; pz = dEdr * uz;
    }
    const uint32_t mask = __ballot_sync(0xffffffffu, isang);
    bool in_table = false;
    if (isang) {
      const int slot = m + __popc(mask & lt);
      if (slot < MAX_ANG) {
        float sn, cs;
        __sincosf((PI_F / RC_A) * r, &sn, &cs);
        S.ur[slot] = make_float4(ux, uy, uz, r);
        S.fs[slot] = make_float4(0.5f * cs + 0.5f, -(PI_F / (2.0f * RC_A)) * sn,
                                 __int_as_float(sp), __int_as_float(e));
        S.pr[slot] = make_float4(px, py, pz, 0.f);
        in_table = true;
      }
    }
    if (e < re && !in_table) {                   // purely radial neighbour: final already
      edge[e] = make_float4(px, py, pz, 0.f);
      sx += px; sy += py; sz += pz;
    }
    m += __popc(mask);
  }
  if (g_pending) cp_async_wait<0>();             // an atom without neighbours
  m = min(m, MAX_ANG);                           // overflow was flagged by K2
  __syncwarp();
  // ---- angular ----
  const int T = (m * (m - 1)) >> 1;
  float Sx[3] = {0.f, 0.f, 0.f}, Sy[3] = {0.f, 0.f, 0.f}, Sz[3] = {0.f, 0.f, 0.f};
  float Sc[3] = {0.f, 0.f, 0.f}, Sr[3] = {0.f, 0.f, 0.f};
  for (int t0 = 0; t0 < T; t0 += K4_TCH) {
    const int nt = min(K4_TCH, T - t0);
    for (int q = lane; q < nt; q += 32) {
      int j, k;
      tri_decode(t0 + q, m, j, k);
      const float4 uj = S.ur[j], uk = S.ur[k];
      const float4 fj = S.fs[j], fk = S.fs[k];
      const float c = COS_SCALE * (uj.x * uk.x + uj.y * uk.y + uj.z * uk.z);
      const float s = sqrtf(fmaf(-c, c, 1.0f));
      const float rbar = 0.5f * (uj.w + uk.w);
      const float* gp = S.gA + GA_STRIDE * pair_block(__float_as_int(fj.z), __float_as_int(fk.z));
      // angular factors two shifts at a time (packed fp32 pairs: half the issue slots)
      float2 A2[NSHF_Z / 2], dA2[NSHF_Z / 2];
      const float2 c2 = make_float2(c, c), s2 = make_float2(s, s), nc2 = make_float2(-c, -c);
      const float2 half2 = make_float2(0.5f, 0.5f), m16 = make_float2(-16.0f, -16.0f);
#pragma unroll
      for (int b = 0; b < NSHF_Z / 2; ++b) {
        const float2 cz = make_float2(c_tab.cos_z[2 * b], c_tab.cos_z[2 * b + 1]);
        const float2 sz_ = make_float2(c_tab.sin_z[2 * b], c_tab.sin_z[2 * b + 1]);
        const float2 q1 = pk_fma(half2, pk_fma(c2, cz, pk_mul(s2, sz_)), half2);
        const float2 q2 = pk_mul(q1, q1), q4 = pk_mul(q2, q2), q8 = pk_mul(q4, q4), q16 = pk_mul(q8, q8);
        A2[b] = pk_mul(q16, q16);
        // dA/dtheta = -16 q^31 sin(theta - theta_b),  sin(theta - theta_b) = s cz - c sz
        const float2 q31 = pk_mul(pk_mul(pk_mul(q16, q8), pk_mul(q4, q2)), q1);
        dA2[b] = pk_mul(pk_mul(q31, m16), pk_fma(s2, cz, pk_mul(nc2, sz_)));
      }
      float G0 = 0.f, Gr = 0.f, Gt = 0.f;
#pragma unroll
      for (int a = 0; a < NSHF_A; ++a) {
        const float4 g0 = *reinterpret_cast<const float4*>(gp + 8 * a);
        const float4 g1 = *reinterpret_cast<const float4*>(gp + 8 * a + 4);
        const float2 ga = make_float2(g0.x, g0.y), gb = make_float2(g0.z, g0.w), gc = make_float2(g1.x, g1.y),
                     gd = make_float2(g1.z, g1.w);
        const float2 u2 = pk_fma(gd, A2[3], pk_fma(gc, A2[2], pk_fma(gb, A2[1], pk_mul(ga, A2[0]))));
        const float2 v2 = pk_fma(gd, dA2[3], pk_fma(gc, dA2[2], pk_fma(gb, dA2[1], pk_mul(ga, dA2[0]))));
        const float ua = u2.x + u2.y, va = v2.x + v2.y;
        const float dr = rbar - c_tab.shf_a[a];
        const float B = ex2_approx(-(ETA_A * LOG2E) * dr * dr);
        const float dB = -2.0f * ETA_A * dr * B;
        G0 = fmaf(ua, B, G0); Gr = fmaf(ua, dB, Gr); Gt = fmaf(va, B, Gt);
      }
      const float fcj = fj.x, fck = fk.x, dfcj = fj.y, dfck = fk.y;
      // dE/dcos(phi) = dE/dtheta * dtheta/dcos(phi),  dtheta/dcos(phi) = -0.95 / sin(theta)
      S.tC[q] = 2.0f * fcj * fck * Gt * (-COS_SCALE / s);
      S.tJ[q] = 2.0f * fck * fmaf(0.5f * Gr, fcj, G0 * dfcj);
      S.tK[q] = 2.0f * fcj * fmaf(0.5f * Gr, fck, G0 * dfck);
    }
    __syncwarp();
    // rows (smaller index j) this chunk of the lexicographic triple order touches: a neighbour n
    // meets only partners j < n with j in [j_lo, j_hi] and, if its own row is among them, the
    // partners k > n whose triple lies in the chunk -- in ascending partner order, as a scan over
    // all partners would, at a cost that does not grow with the number of chunks
    int j_lo = 0, j_hi = m - 2, kk;
    if (T > K4_TCH) {                             // (a single chunk holds every row)
      tri_decode(t0, m, j_lo, kk);
      tri_decode(t0 + nt - 1, m, j_hi, kk);
    }
#pragma unroll
    for (int h = 0; h < 3; ++h) {
      const int n = (int)lane + 32 * h;
      if (n < m) {                                // (h*32 < m is warp-uniform; lanes beyond idle)
        const float4 un = S.ur[n];
        auto meet = [&](int k, int t, float R) {
          const float4 uk = S.ur[k];
          const float C = S.tC[t];
          const float cphi = un.x * uk.x + un.y * uk.y + un.z * uk.z;
          Sx[h] = fmaf(C, uk.x, Sx[h]); Sy[h] = fmaf(C, uk.y, Sy[h]); Sz[h] = fmaf(C, uk.z, Sz[h]);
          Sc[h] = fmaf(C, cphi, Sc[h]);
          Sr[h] += R;
        };
        for (int j = j_lo; j <= min(j_hi, n - 1); ++j) {          // n is the larger index of (j, n)
          const int t = tri_row_start(j, m) + (n - j - 1) - t0;
          if (t >= 0 && t < nt) meet(j, t, S.tK[t]);
        }
        if (n >= j_lo && n <= j_hi) {                             // n is the smaller index of (n, k)
          const int base = tri_row_start(n, m) - (n + 1) - t0;    // t = base + k
          for (int k = max(n + 1, -base); k <= min(m - 1, nt - 1 - base); ++k) meet(k, base + k, S.tJ[base + k]);
        }
      }
    }
    __syncwarp();
  }
#pragma unroll
  for (int h = 0; h < 3; ++h) {
    const int n = (int)lane + 32 * h;
    if (n < m) {
      const float4 un = S.ur[n];
      const float4 pr = S.pr[n];
      const float rinv = 1.0f / un.w;
      const float gx = fmaf(Sr[h], un.x, (Sx[h] - Sc[h] * un.x) * rinv) + pr.x;
      const float gy = fmaf(Sr[h], un.y, (Sy[h] - Sc[h] * un.y) * rinv) + pr.y;
      const float gz = fmaf(Sr[h], un.z, (Sz[h] - Sc[h] * un.z) * rinv) + pr.z;
      edge[__float_as_int(S.fs[n].w)] = make_float4(gx, gy, gz, 0.f);
      sx += gx; sy += gy; sz += gz;
    }
  }
  sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
  if (lane == 0) self[i] = make_float4(sx, sy, sz, 0.f);
}

// K4b: gather.  frc[a] = {F_a, e_a}.
constexpr int K4B_WARPS = 8;
__global__ void __launch_bounds__(K4B_WARPS * 32)
k4b_gather_kernel(int n_atoms, const int* __restrict__ r_off, const int* __restrict__ r_idx, int cap_r,
                  const float4* __restrict__ edge, const float4* __restrict__ self,
                  const int* __restrict__ row_of_atom, const float* __restrict__ e_row,
                  float4* __restrict__ frc) {
  const int a = blockIdx.x * K4B_WARPS + (threadIdx.x >> 5);
  if (a >= n_atoms) return;
  const uint32_t lane = lane_id();
  const int rb = r_off[a];
  // on capacity overflow (flagged by K1) rows at the end are unwritten: outputs unspecified, no wild reads
  const int re = r_off[n_atoms] <= cap_r ? r_off[a + 1] : rb;
  float gx = 0.f, gy = 0.f, gz = 0.f;
  for (int e = rb + (int)lane; e < re; e += 32) {
    const int j = r_idx[e];
    int lo = r_off[j], hi = r_off[j + 1] - 1;     // find a in row j
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (r_idx[mid] < a) lo = mid + 1; else hi = mid;
    }
    const float4 p = edge[lo];
    gx += p.x; gy += p.y; gz += p.z;
  }
  gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz);
  if (lane == 0) {
    const float4 s = self[a];
    frc[a] = make_float4(s.x - gx, s.y - gy, s.z - gz, e_row[row_of_atom[a]]);
  }
}

// per-system potential energy: one CTA per system, fixed-order tree, fp64 partials
// (128 threads for small replicas; 1024 for cell-list systems, whose thousands of atoms would
// otherwise be a long serial chain of loads per thread)
template <int ESUM_THREADS>
__global__ void __launch_bounds__(ESUM_THREADS)
k_energy_sum_kernel(const int* __restrict__ sys_off, const float4* __restrict__ frc,
                    float* __restrict__ E, uint32_t* __restrict__ status) {
  __shared__ double part[ESUM_THREADS];
  const int s = blockIdx.x;
  const int b = sys_off[s], e = sys_off[s + 1];
  double acc = 0.0;
  for (int i = b + threadIdx.x; i < e; i += ESUM_THREADS) acc += (double)frc[i].w;
  part[threadIdx.x] = acc;
  __syncthreads();
  for (int o = ESUM_THREADS / 2; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) part[threadIdx.x] += part[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const float v = (float)part[0];
    E[s] = v;
    if (!isfinite(v)) atomicOr(status, ST_NONFINITE);
  }
}

}  // namespace pfc
