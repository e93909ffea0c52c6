// k4_forces.cuh -- K4: chain rule from g_i = dE/dAEV_i to per-atom forces, with
// fixed-order accumulation (O7; "forces by backprop").
//
// K4a (centre-owned, one warp per atom i): recomputes the pair/triple geometry
// and computes, for every entry e = (i -> j) of atom i's neighbour row,
//      P_e = sum_a g_i[a] * dAEV_i[a]/dx_j        (gradient, not force)
// plus self[i] = sum_e P_e.  By translation invariance dE_i/dx_i = -self[i].
// Brute-force systems: P_e is written where atom j will read it, edge[rev(e)], rev(i -> j) = the position of i in
// row j (rows are symmetric and sorted), found with ONE load from K1's rank table (ballot + running count per
// 32-candidate chunk of j's scan; row and table of j follow from my own by arithmetic, a system's atoms share
// capacity and stride); K4b then reads its row contiguously.  Cell-list systems have no such table: P_e stays in
// my own slot edge[e] and K4b finds rev(e) by binary search in row j.
//   radial : lane <-> entry, 16 shells.
//   angular: the m(m-1)/2 triples of the m angular neighbours (table in row order) are
//            enumerated in round-robin (circulant) order: slot q = (d-1) m + a is the pair
//            {a, (a+d) mod m}, d = 1 .. m/2 -- an order that decodes with one multiply
//            (no square root, no search loop) and whose inverse, which phase 2 needs, is a
//            running index.
//            phase 1, lane <-> slot: the three scalars C = dE/dcos(phi), Ra = dE/dr_a,
//            Rb = dE/dr_b into shared memory, whole rounds d at a time;
//            phase 2, lane <-> angular neighbour n: for every round d of the chunk it meets
//            its partners (n+d) mod m and (n-d) mod m in that fixed order:
//               grad_n = (sum_k C u_k - (sum_k C cos(phi)) u_n)/r_n + (sum_k R) u_n.
// K4b (one warp per atom a):
//      F_a = self[a] - sum_{k < cnt(a), ascending} P_(j_k -> a),   j_k = k-th neighbour of a,
// read from slot k of a's own row (brute-force systems) or from edge[rev(a -> j_k)] (cell-list systems).
// Every slot has exactly one writer and the summation order is fixed.  No float atomics anywhere.
#pragma once
#include "aev_common.cuh"

namespace pfc {

constexpr int K4_TCH = 128;              // triple slots per shared-memory pass (>= MAX_ANG: at least one round)
constexpr int GA_STRIDE = 36;            // padded stride of one 32-float g block
static_assert(K4_TCH >= MAX_ANG, "a chunk holds at least one whole round of the circulant order");

struct AevBwdSmem {
  float4 ur[MAX_ANG];                    // unit vector, r
  float4 fs[MAX_ANG];                    // fc, dfc (RC_A), species bits, entry index bits
  float4 pr[MAX_ANG];                    // radial part of P for this neighbour
  float gR[RAD_LEN];
  float gA[NPAIR * GA_STRIDE];
  float tC[K4_TCH], tA[K4_TCH], tB[K4_TCH];
};

#ifndef PFC_K4A_MINB
#define PFC_K4A_MINB 25
#endif
__global__ void __launch_bounds__(AEV_WARPS * 32, PFC_K4A_MINB)
k4a_aev_bwd_kernel(int n_atoms, const float4* __restrict__ xs, const float4* __restrict__ xsl,
                   const int* __restrict__ row_beg, const uint32_t* __restrict__ nbr, const int2* __restrict__ cnt,
                   const int* __restrict__ row_of_atom, const int4* __restrict__ rank_info,
                   const int2* __restrict__ rank_tab,
                   const float* __restrict__ g, float4* __restrict__ edge, float4* __restrict__ self) {
  __shared__ __align__(16) AevBwdSmem sm[AEV_WARPS];
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
  const int rb = row_beg[i];
  const int re = rb + cnt[i].x;
  // Atoms of one brute-force system share the row capacity and the rank-table stride, so neighbour j's row and
  // table follow from my own by arithmetic: the lookup is ONE load.  Cell-list systems (no table): tab_i < 0.
  const int4 ri = rank_info[i];                  // {my first table word or -1, first atom of my system, words per atom, -}
  const int rel_i = i - ri.y;                    // my index inside my system
  const int tab_i = ri.x, words_i = ri.z;
  const int cap_i = row_beg[i + 1] - rb;
  int m = 0;
  float sx = 0.f, sy = 0.f, sz = 0.f;            // this lane's share of self[i]
  for (int c0 = rb; c0 < re; c0 += 32) {
    int e = c0 + (int)lane;                      // my entry; from the lookup below on: the slot its gradient goes to
    const bool live = e < re;
    NbrGeom ng;
    ng.ang = false; ng.sp = 0; ng.r = 1.0f; ng.ux = ng.uy = ng.uz = 0.0f;
    float px = 0.f, py = 0.f, pz = 0.f;
    float fc = 0.f, dfc = 0.f;
    if (live) {
      const uint32_t w = nbr[e];
      if (tab_i >= 0) {
        // rev(e): where neighbour j keeps me in ITS row
        const int dj = nbr_index(w) - i;
        const int2 t = rank_tab[tab_i + dj * words_i + (rel_i >> 5)];
        // (on a row-capacity overflow, flagged by K1, outputs are unspecified -- but the slot stays inside row j)
        e = rb + dj * cap_i + min(t.y + __popc((uint32_t)t.x & ((1u << (rel_i & 31)) - 1u)), cap_i - 1);
      }                                          // (cell-list system: the gradient stays in my own slot, K4b searches)
      ng = nbr_geometry(w, xi, li, xs, xsl);
      float sn, cs;
      __sincosf((PI_F / RC_R) * ng.r, &sn, &cs);
      fc = 0.5f * cs + 0.5f; dfc = -(PI_F / (2.0f * RC_R)) * sn;
    }
    if (g_pending) {                             // warp-uniform: every lane's granules, then the handover
      cp_async_wait<0>();
      __syncwarp();
      g_pending = false;
    }
    if (live) {
      // two shells at a time in packed fp32 pairs (the exponentials stay scalar SFU calls)
      const float2* gs = reinterpret_cast<const float2*>(S.gR + NSHF_R * ng.sp);
      const float2 r2 = make_float2(ng.r, ng.r), m1 = make_float2(-1.0f, -1.0f), fc2 = make_float2(fc, fc),
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
      px = dEdr * ng.ux; py = dEdr * ng.uy; pz = dEdr * ng.uz;
    }
    const uint32_t mask = __ballot_sync(0xffffffffu, ng.ang);
    bool in_table = false;
    if (ng.ang) {
      const int slot = m + __popc(mask & lt);
      if (slot < MAX_ANG) {
        float sn, cs;
        __sincosf((PI_F / RC_A) * ng.r, &sn, &cs);
        S.ur[slot] = make_float4(ng.ux, ng.uy, ng.uz, ng.r);
        S.fs[slot] = make_float4(0.5f * cs + 0.5f, -(PI_F / (2.0f * RC_A)) * sn,
                                 __int_as_float(ng.sp), __int_as_float(e));
        S.pr[slot] = make_float4(px, py, pz, ng.rinv);
        in_table = true;
      }
    }
    if (live && !in_table) {                     // purely radial neighbour: final already
      edge[e] = make_float4(px, py, pz, 0.f);
      sx += px; sy += py; sz += pz;
    }
    m += __popc(mask);
  }
  if (g_pending) cp_async_wait<0>();             // an atom without neighbours
  m = min(m, MAX_ANG);                           // overflow was flagged by K2
  __syncwarp();
  // ---- angular ----
  // rounds d = 1 .. m/2; round d holds the m pairs {a, (a+d) mod m}, except the last round of an
  // even m (d = m/2), which holds only a < m/2.  T = m(m-1)/2 slots in all.
  const int T = (m * (m - 1)) >> 1;
  const int rounds = m >> 1;                     // (m odd: (m-1)/2 full rounds; m even: m/2 - 1 full + one half round)
  const int rpc = m > 0 ? K4_TCH / m : 1;        // whole rounds per chunk (>= 1)
  float Sx[3] = {0.f, 0.f, 0.f}, Sy[3] = {0.f, 0.f, 0.f}, Sz[3] = {0.f, 0.f, 0.f};
  float Sc[3] = {0.f, 0.f, 0.f}, Sr[3] = {0.f, 0.f, 0.f};
  for (int d0 = 1; d0 <= rounds; d0 += rpc) {    // chunk = rounds d0 .. d0 + rpc - 1
    const int t0 = (d0 - 1) * m;
    const int nt = min(rpc * m, T - t0);
    for (int q = lane; q < nt; q += 32) {
      const int dd = small_div(q, m);            // round d0 + dd
      const int a = q - dd * m;
      int b = a + d0 + dd;
      b = b >= m ? b - m : b;
      const float4 ua = S.ur[a], ub = S.ur[b];
      const float4 fa = S.fs[a], fb = S.fs[b];
      const float c = COS_SCALE * (ua.x * ub.x + ua.y * ub.y + ua.z * ub.z);
      const float s = sqrt_newton(fmaf(-c, c, 1.0f));
      const float rbar = 0.5f * (ua.w + ub.w);
      const float* gp = S.gA + GA_STRIDE * pair_block(__float_as_int(fa.z), __float_as_int(fb.z));
      // angular factors two shifts at a time (packed fp32 pairs: half the issue slots)
      float2 A2[NSHF_Z / 2], dA2[NSHF_Z / 2];
      const float2 c2 = make_float2(c, c), s2 = make_float2(s, s), nc2 = make_float2(-c, -c);
      const float2 half2 = make_float2(0.5f, 0.5f), m16 = make_float2(-16.0f, -16.0f);
#pragma unroll
      for (int z = 0; z < NSHF_Z / 2; ++z) {
        const float2 cz = make_float2(c_tab.cos_z[2 * z], c_tab.cos_z[2 * z + 1]);
        const float2 sz_ = make_float2(c_tab.sin_z[2 * z], c_tab.sin_z[2 * z + 1]);
        const float2 q1 = pk_fma(half2, pk_fma(c2, cz, pk_mul(s2, sz_)), half2);
        const float2 q2 = pk_mul(q1, q1), q4 = pk_mul(q2, q2), q8 = pk_mul(q4, q4), q16 = pk_mul(q8, q8);
        A2[z] = pk_mul(q16, q16);
        // dA/dtheta = -16 q^31 sin(theta - theta_b),  sin(theta - theta_b) = s cz - c sz
        const float2 q31 = pk_mul(pk_mul(pk_mul(q16, q8), pk_mul(q4, q2)), q1);
        dA2[z] = pk_mul(pk_mul(q31, m16), pk_fma(s2, cz, pk_mul(nc2, sz_)));
      }
      float G0 = 0.f, Gr = 0.f, Gt = 0.f;
#pragma unroll
      for (int sa = 0; sa < NSHF_A; ++sa) {
        const float4 g0 = *reinterpret_cast<const float4*>(gp + 8 * sa);
        const float4 g1 = *reinterpret_cast<const float4*>(gp + 8 * sa + 4);
        const float2 ga = make_float2(g0.x, g0.y), gb = make_float2(g0.z, g0.w), gc = make_float2(g1.x, g1.y),
                     gd = make_float2(g1.z, g1.w);
        const float2 u2 = pk_fma(gd, A2[3], pk_fma(gc, A2[2], pk_fma(gb, A2[1], pk_mul(ga, A2[0]))));
        const float2 v2 = pk_fma(gd, dA2[3], pk_fma(gc, dA2[2], pk_fma(gb, dA2[1], pk_mul(ga, dA2[0]))));
        const float uu = u2.x + u2.y, vv = v2.x + v2.y;
        const float dr = rbar - c_tab.shf_a[sa];
        const float B = ex2_approx(-(ETA_A * LOG2E) * dr * dr);
        const float dB = -2.0f * ETA_A * dr * B;
        G0 = fmaf(uu, B, G0); Gr = fmaf(uu, dB, Gr); Gt = fmaf(vv, B, Gt);
      }
      const float fca = fa.x, fcb = fb.x, dfca = fa.y, dfcb = fb.y;
      // dE/dcos(phi) = dE/dtheta * dtheta/dcos(phi),  dtheta/dcos(phi) = -0.95 / sin(theta)
      S.tC[q] = 2.0f * fca * fcb * Gt * (-COS_SCALE * rcp_approx(s) * fmaf(-s, rcp_approx(s), 2.0f));
      S.tA[q] = 2.0f * fcb * fmaf(0.5f * Gr, fca, G0 * dfca);
      S.tB[q] = 2.0f * fca * fmaf(0.5f * Gr, fcb, G0 * dfcb);
    }
    __syncwarp();
    const int nr = min(rpc, rounds - d0 + 1);    // rounds in this chunk
#pragma unroll
    for (int h = 0; h < 3; ++h) {
      const int n = (int)lane + 32 * h;
      if (n < m) {                               // (h*32 < m is warp-uniform; lanes beyond idle)
        const float4 un = S.ur[n];
        auto meet = [&](int k, float C, float R) {
          const float4 uk = S.ur[k];
          const float cphi = un.x * uk.x + un.y * uk.y + un.z * uk.z;
          Sx[h] = fmaf(C, uk.x, Sx[h]); Sy[h] = fmaf(C, uk.y, Sy[h]); Sz[h] = fmaf(C, uk.z, Sz[h]);
          Sc[h] = fmaf(C, cphi, Sc[h]);
          Sr[h] += R;
        };
        int k1 = n + d0, k2 = n - d0;            // partners of round d0: (n + d) mod m and (n - d) mod m
        k1 = k1 >= m ? k1 - m : k1;
        k2 = k2 < 0 ? k2 + m : k2;
        for (int r = 0; r < nr; ++r) {
          const int d = d0 + r, base = r * m;
          const bool half_round = 2 * d == m;    // pairs {a, a + m/2}, a < m/2 only
          if (!half_round || n < d) meet(k1, S.tC[base + n], S.tA[base + n]);      // I am a of the pair
          if (!half_round || n >= d) meet(k2, S.tC[base + k2], S.tB[base + k2]);   // I am b of the pair {k2, n}
          k1 = k1 + 1 >= m ? k1 + 1 - m : k1 + 1;
          k2 = k2 - 1 < 0 ? k2 - 1 + m : k2 - 1;
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
      const float rinv = pr.w;
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

// K4b: gather.  frc[a] = {F_a, e_a}.  EIGHT lanes per atom, four atoms per warp: a row has 27 entries on
// average and the kernel is a short chain of dependent loads per atom -- four atoms per warp put four times as
// many chains in flight (64 -> 43 us on config 4 against one warp per atom).
constexpr int K4B_WARPS = 8, K4B_LANES = 8, K4B_ATOMS = K4B_WARPS * 32 / K4B_LANES;
__global__ void __launch_bounds__(K4B_WARPS * 32)
k4b_gather_kernel(int n_atoms, const int* __restrict__ row_beg, const uint32_t* __restrict__ nbr,
                  const int2* __restrict__ cnt, const int4* __restrict__ rank_info,
                  const float4* __restrict__ edge, const float4* __restrict__ self,
                  const int* __restrict__ row_of_atom, const float* __restrict__ e_row,
                  float4* __restrict__ frc) {
  const int a = blockIdx.x * K4B_ATOMS + (int)(threadIdx.x / K4B_LANES);
  const int sub = (int)(threadIdx.x % K4B_LANES);
  const bool have = a < n_atoms;                    // (no early return: the shuffles below take the whole warp)
  int rb = 0, re = 0;
  bool own_row = true;
  float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
  float ea = 0.f;
  if (have) {
    rb = row_beg[a];
    re = rb + cnt[a].x;
    own_row = rank_info[a].x >= 0;                  // brute-force system: my neighbours wrote into my row
    // (requested now, used at the end: they do not wait for the row)
    s = self[a];
    ea = e_row[row_of_atom[a]];
  }
  float gx = 0.f, gy = 0.f, gz = 0.f;
  for (int e = rb + sub; e < re; e += K4B_LANES) {
    int slot = e;
    if (!own_row) {
      // find a in row j (on a row-capacity overflow, flagged by K1, the entry may be missing: outputs
      // are unspecified then, but the search stays inside row j)
      const int j = nbr_index(nbr[e]);
      int lo = row_beg[j], hi = lo + max(cnt[j].x, 1) - 1;
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (nbr_index(nbr[mid]) < a) lo = mid + 1; else hi = mid;
      }
      slot = lo;
    }
    const float4 p = edge[slot];
    gx += p.x; gy += p.y; gz += p.z;
  }
#pragma unroll
  for (int o = K4B_LANES / 2; o > 0; o >>= 1) {     // fixed xor tree inside the atom's eight lanes: deterministic
    gx += __shfl_xor_sync(0xffffffffu, gx, o);
    gy += __shfl_xor_sync(0xffffffffu, gy, o);
    gz += __shfl_xor_sync(0xffffffffu, gz, o);
  }
  if (have && sub == 0) frc[a] = make_float4(s.x - gx, s.y - gy, s.z - gz, ea);
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
