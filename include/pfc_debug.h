/* pfc_debug.h -- measurement and debug entry points of libpfc, kept out of the provider
 * boundary pfc.h ("keep them few").  bench.py and the tests use them; an MD
 * engine driving the potential never needs them. */
#ifndef PFC_DEBUG_H_
#define PFC_DEBUG_H_

#include "pfc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement (per-kernel roofline): the same kernel sequence as
 * pfc_energy_forces, launched kernel by kernel with a CUDA event recorded on `stream` at every
 * stage boundary; synchronises and returns the device time of each stage in milliseconds,
 * ms HOST [PFC_N_STAGES]: 0 = K1 neighbour build, 1 = K2 AEV forward, 2 = K3 MLP
 * forward+backward, 3 = K4a AEV backward, 4 = K4b force gather, 5 = per-system energy sum,
 * 6 = K5, the fused integrator kernel of a steady-state step (run on internal staging buffers: the
 * caller's state does not move; 0 while a pfc_run_host state occupies those buffers). */
#define PFC_N_STAGES 7
int pfc_profile_stages(pfc_t *ctx, const float *pos, float *E, float *F, void *stream, float *ms);

/* Work counts of the last evaluation, for the roofline arithmetic: counts HOST [5] =
 * {radial row entries, angular row entries, triples (sum over atoms of m(m-1)/2, m = angular
 * neighbours), brute-force distance tests per evaluation, candidate-row builds of the cell-list
 * systems since pfc_create (skin list: far fewer than evaluations)}.  Synchronises the handle's stream. */
int pfc_work_counts(pfc_t *ctx, int64_t *counts);

/* Timeline of the tensor-core MLP kernel (one relaunch of K3 on the AEV rows of the last evaluation; the
 * outputs it rewrites are unchanged): SM clock values recorded by the first CTA at the scheduling events of
 * its first 8 tile iterations, 128 slots per iteration (slot meaning: TC_TRACE comment in csrc/k3_mlp_tc.cuh);
 * 0 = event not reached.  cycles HOST [n], n <= 1024.  PFC_ERR_STATE on the FP32 path.  Synchronises. */
int pfc_k3_timeline(pfc_t *ctx, int64_t *cycles, int32_t n);

/* Parity helper: synchronous cudaMemcpy of `bytes` from a DEVICE pointer returned by the
 * getters of pfc.h into HOST memory. */
int pfc_copy_to_host(const void *device_src, void *host_dst, size_t bytes);

/* How the tensor core accumulates: ONE accumulator chain of n_mma tcgen05.mma
 * kind::f16 instructions (M 128, N 64, K 16, fp32 accumulate), instruction i multiplying the 16-k slice
 * (i mod n_slices) of A DEVICE [128][16 n_slices] and B DEVICE [64][16 n_slices] (row-major fp32 values, which
 * must be exactly representable in fp16; 1 <= n_slices <= 16), staged in shared memory exactly as the MLP
 * kernel stages its operands.  D DEVICE [128][64]: the raw accumulator.  No handle; enqueues one kernel on
 * `stream` of the current device. */
int pfc_tc_chain_probe(const float *A, const float *B, int32_t n_slices, int32_t n_mma, float *D, void *stream);

/* Truncation compensation of the tensor-core MLP, per element e = 0..3:
 * out HOST [32], out[8e + ..] = {lambda forward, lambda backward, residual slope of e_i, residual slope of g,
 * max|de| / rms e, max|dg| / rms g (all against the library's FP32 MLP on the calibration batch; 0 for an
 * element below the calibration size), 1 if the scales are final (calibrated or fixed by pfc_tuning_t),
 * 1 if PFC_MLP_AUTO went back to the FP32 MLP because an element missed the check}. */
int pfc_tc_calibration(pfc_t *ctx, float *out);

/* The MLP path in use (PFC_MLP_AUTO resolved by pfc_create; after the first evaluation: by the
 * calibration check as well). */
int pfc_mlp_path(pfc_t *ctx, int32_t *path);

/* Kernel launches one energy/forces evaluation and one steady-state MD step consist of, and the
 * number of MD steps pfc_step captures per CUDA graph. */
int pfc_launch_counts(pfc_t *ctx, int32_t *per_energy_forces, int32_t *per_step, int32_t *steps_per_graph);

#ifdef __cplusplus
}
#endif
#endif /* PFC_DEBUG_H_ */
