// pfc_common.cuh -- model constants, device-side views and small helpers shared
// by the pfc kernels (sm_100a).  Nothing here is shared with oracle/.
//
// Constants restate DESIGN.md "Model constants" (readings S2-S8): every model
// constant is DEFINED as an fp32 value.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pfc {

constexpr int NSPEC = 4;
constexpr int NSHF_R = 16, NSHF_A = 4, NSHF_Z = 8, NPAIR = 10;
constexpr int RAD_LEN = NSPEC * NSHF_R;            // 64
constexpr int ANG_LEN = NPAIR * NSHF_A * NSHF_Z;   // 320
constexpr int AEV_LEN = RAD_LEN + ANG_LEN;         // 384
constexpr int D0 = AEV_LEN, D1 = 160, D2 = 128, D3 = 96;
constexpr int W_PER_ELEM = D1 * D0 + D1 + D2 * D1 + D2 + D3 * D2 + D3 + D3 + 1;  // 94,689
constexpr int ROW_PAD = 128;                       // element blocks padded to this many rows
constexpr int MAX_ANG = 96;                        // PFC_MAX_ANGULAR
constexpr int BRUTE_MAX = 2048;                    // systems above this use the cell list

constexpr float RC2_R = 27.04f;                    // S6: 0x41d851ec (not 5.2f*5.2f)
constexpr float RC2_A = 12.25f;
constexpr float RC_R = 5.2f, RC_A = 3.5f;
constexpr float ETA_R = 16.0f, ETA_A = 8.0f;
constexpr float COS_SCALE = 0.95f;                 // S5
constexpr float CELU_ALPHA = 0.1f;
constexpr float PI_F = 3.14159265358979323846f;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float ACC_F = 9.648533216e-3f;           // (A/fs^2) per (eV/A/amu)

// device status bits (mirror include/pfc.h)
constexpr uint32_t ST_RADIAL_OVERFLOW = 1u, ST_ANGULAR_OVERFLOW = 2u, ST_ANGULAR_ROW = 4u,
                   ST_NONFINITE = 8u, ST_CELL_OVERFLOW = 16u;

// Model tables in constant memory: compile-time constants, identical for every handle (nothing
// per-handle lives in constant memory; the masses are in StepParams).
//   shf_r[k] = (float)(0.9 + k*0.26875)  (S2);  shf_a = 0.9, 1.55, 2.2, 2.85  (S3);
//   cos_z[b], sin_z[b] = (float)cos / sin of (double)(float)SHF_Z[b], SHF_Z = 0.19634954 + b*pi/8 as
//   the fp32 literals of DESIGN.md (S3, S8).
struct ModelTables {
  float shf_r[NSHF_R];
  float shf_a[NSHF_A];
  float cos_z[NSHF_Z];
  float sin_z[NSHF_Z];
};
__constant__ ModelTables c_tab = {
    {0.9f, 1.16875f, 1.4375f, 1.70625f, 1.975f, 2.24375f, 2.5125f, 2.78125f,
     3.05f, 3.31875f, 3.5875f, 3.85625f, 4.125f, 4.39375f, 4.6625f, 4.93125f},
    {0.9f, 1.55f, 2.2f, 2.85f},
    {0.9807852506637573f, 0.8314695954322815f, 0.5555702447891235f, 0.19509035348892212f,
     -0.19509032368659973f, -0.5555701851844788f, -0.8314696550369263f, -0.9807853102684021f},
    {0.19509032368659973f, 0.5555702447891235f, 0.8314695954322815f, 0.9807852506637573f,
     0.9807852506637573f, 0.8314696550369263f, 0.5555701851844788f, 0.19509030878543854f}};

// Neighbour-row entry word (internal format of K1's rows): bits 0..28 neighbour index j,
// bits 29..30 species of j, bit 31 set when j is also an angular neighbour (d2 < RC2_A).
constexpr uint32_t NBR_IDX_MASK = 0x1FFFFFFFu;
__device__ __forceinline__ int nbr_index(uint32_t w) { return (int)(w & NBR_IDX_MASK); }
__device__ __forceinline__ int nbr_species(uint32_t w) { return (int)((w >> 29) & 3u); }
__device__ __forceinline__ bool nbr_angular(uint32_t w) { return (w >> 31) != 0u; }

// Step parameters live in device memory so a captured graph is reusable for any dt.
struct StepParams {
  float dt;        // fs
  float half_dt;   // dt/2
  float inv_mass_acc[NSPEC];  // ACC / m_s of THIS handle (pfc_desc_t.masses_amu)
  // Langevin (O9): v <- c1 v + sigma[species] xi,  sigma_s = c2 sqrt(kB T ACC / m_s)
  float c1;
  float sigma[NSPEC];
  uint32_t seed_lo, seed_hi;
  uint32_t step;   // Langevin steps taken since pfc_set_state: counter word 1 of the generator
  uint32_t ticket; // blocks of the running Langevin kernel that have finished (last one advances step)
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// O2 predicate: three subtractions, three products, two sums, each rounded to
// nearest fp32, never contracted into FMAs (S6).
__device__ __forceinline__ float dist2_rn(float ax, float ay, float az, float bx, float by, float bz) {
  float dx = __fsub_rn(ax, bx), dy = __fsub_rn(ay, by), dz = __fsub_rn(az, bz);
  float s = __fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy));
  return __fadd_rn(s, __fmul_rn(dz, dz));
}

// species-pair block of the angular AEV: HH0 HC1 HN2 HO3 CC4 CN5 CO6 NN7 NO8 OO9
__device__ __forceinline__ int pair_block(int za, int zb) {
  int s1 = min(za, zb), s2 = max(za, zb);
  return s1 * NSPEC - ((s1 * (s1 - 1)) >> 1) + (s2 - s1);
}

// Packed fp32 pairs (sm_100: SASS FFMA2 / FMUL2): one issue slot for two lanes of arithmetic.
__device__ __forceinline__ float2 pk_fma(float2 a, float2 b, float2 c) {
  unsigned long long ua = *reinterpret_cast<unsigned long long*>(&a), ub = *reinterpret_cast<unsigned long long*>(&b),
                     uc = *reinterpret_cast<unsigned long long*>(&c), ud;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
  return *reinterpret_cast<float2*>(&ud);
}
__device__ __forceinline__ float2 pk_mul(float2 a, float2 b) {
  unsigned long long ua = *reinterpret_cast<unsigned long long*>(&a), ub = *reinterpret_cast<unsigned long long*>(&b), ud;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(ud) : "l"(ua), "l"(ub));
  return *reinterpret_cast<float2*>(&ud);
}

// Ampere-style asynchronous 16-byte copies global -> shared (L2 only, no L1 allocation)
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

__device__ __forceinline__ float warp_sum(float v) {   // fixed xor tree: deterministic
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace pfc
