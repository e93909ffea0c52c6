// k0_units.cuh -- unit / layout conversion kernels of the provider-style entry point
// pfc_energy_forces_nm: the paper's callback receives positions in nm and
// returns kJ/mol and kJ/mol/nm (OpenMM units); the hot path works
// in A, eV, eV/A on float4 rows.  1 nm = 10 A, 1 eV = 96.485332 kJ/mol.
#pragma once
#include "pfc_common.cuh"

namespace pfc {

constexpr float NM_TO_A = 10.0f;
constexpr float EV_TO_KJMOL = 96.485332f;
constexpr int K0_THREADS = 256;

// pos_nm [N][3] packed -> float4 {x, y, z, 0} in A
__global__ void __launch_bounds__(K0_THREADS)
k0_pack_nm_kernel(int n_atoms, const float* __restrict__ pos_nm, float4* __restrict__ pos) {
  const int i = blockIdx.x * K0_THREADS + threadIdx.x;
  if (i >= n_atoms) return;
  pos[i] = make_float4(NM_TO_A * pos_nm[3 * i], NM_TO_A * pos_nm[3 * i + 1], NM_TO_A * pos_nm[3 * i + 2], 0.0f);
}

// frc {F, e_i} eV/A, E eV  ->  F [N][3] kJ/mol/nm (optional), E kJ/mol
__global__ void __launch_bounds__(K0_THREADS)
k0_unpack_kj_kernel(int n_atoms, int n_systems, const float4* __restrict__ frc, const float* __restrict__ E,
                    float* __restrict__ F_kj_nm, float* __restrict__ E_kj) {
  const int i = blockIdx.x * K0_THREADS + threadIdx.x;
  if (i < n_systems) E_kj[i] = EV_TO_KJMOL * E[i];
  if (i >= n_atoms || !F_kj_nm) return;
  const float4 f = frc[i];
  const float k = EV_TO_KJMOL * NM_TO_A;
  F_kj_nm[3 * i] = k * f.x; F_kj_nm[3 * i + 1] = k * f.y; F_kj_nm[3 * i + 2] = k * f.z;
}

}  // namespace pfc
