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
  const float kick = (MODE == 2 ? dt : sp->half_dt) * c_tab.inv_mass_acc[species[i]];
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

}  // namespace pfc
