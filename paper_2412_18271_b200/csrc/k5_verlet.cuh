// k5_verlet.cuh -- K5: velocity-Verlet (O8; PAPER.md:73 NVE, fixed step).
//   a = F * ACC / m;  v += dt/2 a;  x += dt v;  [forces];  v += dt/2 a
// fp32 velocities; positions are a two-float sum (x_hi in the caller's buffer,
// x_lo internal), reading S15: one ulp of a 36 A coordinate is 3.8e-6 A, which
// would otherwise eat a fifth of the 1e-4 A trajectory budget in 100 steps.
// The .w lanes of pos/vel are carried through unchanged.
#pragma once
#include "pfc_common.cuh"

namespace pfc {

constexpr int K5_THREADS = 256;

// MODE 0: trailing half kick only.  MODE 1: leading half kick + drift.
// MODE 2: trailing half kick of step n fused with the leading half kick + drift of step n+1.
template <int MODE>
__global__ void __launch_bounds__(K5_THREADS)
k5_verlet_kernel(int n_atoms, const StepParams* __restrict__ sp, const int* __restrict__ species,
                 const float4* __restrict__ frc, float4* __restrict__ pos, float4* __restrict__ vel,
                 float4* __restrict__ xlo) {
  const int i = blockIdx.x * K5_THREADS + threadIdx.x;
  if (i >= n_atoms) return;
  const float dt = sp->dt;
  const float kick = (MODE == 2 ? dt : sp->half_dt) * sp->inv_mass_acc[species[i]];
  const float4 f = frc[i];
  float4 v = vel[i];
  v.x = fmaf(kick, f.x, v.x); v.y = fmaf(kick, f.y, v.y); v.z = fmaf(kick, f.z, v.z);
  vel[i] = v;
  if (MODE == 0) return;
  float4 x = pos[i], lo = xlo[i];
  auto two_sum = [](float& hi, float& l, float add) {
    const float y = add + l;
    const float t = hi + y;
    const float bp = t - hi;
    l = (hi - (t - bp)) + (y - bp);
    hi = t;
  };
  two_sum(x.x, lo.x, dt * v.x);
  two_sum(x.y, lo.y, dt * v.y);
  two_sum(x.z, lo.z, dt * v.z);
  pos[i] = x;
  xlo[i] = lo;
}

__global__ void k5_set_params_kernel(StepParams* sp, float dt) {
  sp->dt = dt;
  sp->half_dt = 0.5f * dt;
}

// ---- Langevin dynamics, BAOAB (O9, readings S27/S28; PAPER.md:94 protocol) ----
// Philox4x32-10, counter (atom, step, 0, 0), key (seed_lo, seed_hi): the same generator the
// oracle implements on its side (no shared code).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t lo0 = 0xD2511F53u * c.x, hi0 = __umulhi(0xD2511F53u, c.x);
    const uint32_t lo1 = 0xCD9E8D57u * c.z, hi1 = __umulhi(0xCD9E8D57u, c.z);
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}
__device__ __forceinline__ float u24(uint32_t w) { return fmaf((float)(w >> 8), 5.9604644775390625e-8f, 2.98023223876953125e-8f); }

__global__ void k5_set_langevin_kernel(StepParams* sp, float c1, float c2, float kT, uint32_t seed_lo,
                                       uint32_t seed_hi) {
  sp->c1 = c1;
  for (int s = 0; s < NSPEC; ++s) sp->sigma[s] = c2 * sqrtf(kT * sp->inv_mass_acc[s]);   // kT in eV
  sp->seed_lo = seed_lo; sp->seed_hi = seed_hi;
}
__global__ void k5_reset_counter_kernel(StepParams* sp) { sp->step = 0; sp->ticket = 0; }

// MODE 1: B(dt/2) A O A.  MODE 2: trailing B(dt/2) of step n fused with B(dt/2) A O A of step n+1.
// (The last trailing half kick is k5_verlet_kernel<0>.)  The step counter lives in device memory so
// the captured graph is replayable; the last block to finish advances it.
template <int MODE>
__global__ void __launch_bounds__(K5_THREADS)
k5_langevin_kernel(int n_atoms, StepParams* __restrict__ sp, const int* __restrict__ species,
                   const float4* __restrict__ frc, float4* __restrict__ pos, float4* __restrict__ vel,
                   float4* __restrict__ xlo) {
  const int i = blockIdx.x * K5_THREADS + threadIdx.x;
  const uint32_t step = sp->step + 1u;
  if (i < n_atoms) {
    const int z = species[i];
    const float dt = sp->dt, hdt = sp->half_dt;
    const float kick = (MODE == 2 ? dt : hdt) * sp->inv_mass_acc[z];
    const float4 f = frc[i];
    float4 v = vel[i];
    v.x = fmaf(kick, f.x, v.x); v.y = fmaf(kick, f.y, v.y); v.z = fmaf(kick, f.z, v.z);      // B
    float4 x = pos[i], lo = xlo[i];
    auto two_sum = [](float& hi, float& l, float add) {
      const float y = add + l;
      const float t = hi + y;
      const float bp = t - hi;
      l = (hi - (t - bp)) + (y - bp);
      hi = t;
    };
    two_sum(x.x, lo.x, hdt * v.x); two_sum(x.y, lo.y, hdt * v.y); two_sum(x.z, lo.z, hdt * v.z);   // A
    const uint4 w = philox4x32_10(make_uint4((uint32_t)i, step, 0u, 0u), make_uint2(sp->seed_lo, sp->seed_hi));
    const float r0 = sqrtf(-2.0f * logf(u24(w.x))), r1 = sqrtf(-2.0f * logf(u24(w.z)));
    float s0, c0, s1, c1v;
    sincospif(2.0f * u24(w.y), &s0, &c0);
    sincospif(2.0f * u24(w.w), &s1, &c1v);
    const float c1 = sp->c1, sg = sp->sigma[z];
    v.x = fmaf(c1, v.x, sg * (r0 * c0)); v.y = fmaf(c1, v.y, sg * (r0 * s0)); v.z = fmaf(c1, v.z, sg * (r1 * c1v));   // O
    two_sum(x.x, lo.x, hdt * v.x); two_sum(x.y, lo.y, hdt * v.y); two_sum(x.z, lo.z, hdt * v.z);   // A
    vel[i] = v; pos[i] = x; xlo[i] = lo;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(&sp->ticket, 1u) == gridDim.x - 1) {   // every block has read sp->step by now
      sp->ticket = 0;
      sp->step = step;
      __threadfence();
    }
  }
}

}  // namespace pfc
