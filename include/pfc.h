/* pfc.h -- C ABI of libpfc: per-step energy, forces and velocity-Verlet update
 * of an ANI-style machine-learned interatomic potential on one NVIDIA B200
 * (sm_100a).
 *
 * What the calls are.  The paper (arxiv 2412.18271, "OpenMM-Python-Force")
 * states the problem: an MD integrator calls a provider every step with the
 * positions and receives the scalar energy, forces being -dE/dx by
 * differentiation (section 2.1 / listing) or returned
 * explicitly (section 3.2); tensors stay on the device
 * (abstract); integration is NVE from 300 K velocities
 * (section 3.1).  BASELINE.json:north_star names the four entry
 * points (pfc_create, pfc_energy_forces, pfc_step, pfc_destroy); the
 * potential itself is BASELINE.json:configs[0] completed by DESIGN.md
 * "Readings" S1-S24.
 *
 * Conventions
 *  - Units: Angstrom, eV, eV/Angstrom, amu, fs, Angstrom/fs.
 *    (OpenMM side of the paper: 1 nm = 10 A, 1 eV = 96.485332 kJ/mol.)
 *  - "DEVICE" pointers are CUDA device memory owned by the caller (PyTorch in
 *    this repository); "HOST" pointers are ordinary host memory.  The library
 *    never allocates device memory: everything it needs is carved out of the
 *    caller's `workspace`.
 *  - pos / vel / frc are arrays of 4 floats per atom (float4, 16-byte
 *    aligned): pos = {x,y,z,ignored}, vel = {vx,vy,vz,ignored},
 *    frc = {Fx,Fy,Fz,e_i} where e_i is the atom's energy contribution.
 *    The .w lanes of caller-owned pos/vel are never written.
 *  - Atoms of system s are the contiguous range sys_offsets[s]..sys_offsets[s+1];
 *    there are no pairs across systems.
 *  - Every call except create/destroy/status/run_host only ENQUEUES work on
 *    the given stream and returns; it never synchronises.  One exception, once per
 *    handle: the FIRST evaluation (pfc_energy_forces, pfc_energy_forces_nm or pfc_step)
 *    of a handle on the tensor-core MLP measures its truncation compensation on that
 *    batch against the library's FP32 MLP (five extra MLP launches)
 *    and synchronises the stream; it must not be issued under a stream capture of the
 *    caller's.  Under PFC_MLP_AUTO the handle stays on the tensor-core MLP only if the
 *    check of that measurement passes (pfc_mlp_path in pfc_debug.h reports the outcome).
 *  - Return value: PFC_OK (0) or a negative PFC_ERR_* code.  Nothing throws or
 *    aborts across this boundary.  Conditions detected on the device
 *    (neighbour capacity overflow, angular row longer than PFC_MAX_ANGULAR,
 *    non-finite energy) set sticky bits readable with pfc_status(); outputs
 *    are then unspecified.
 *  - One handle = one stream = one caller at a time; several handles (with their own
 *    masses, weights and systems) may be live at once.
 *  - Measurement and debug entry points are declared in pfc_debug.h.
 */
#ifndef PFC_H_
#define PFC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PFC_OK 0
#define PFC_ERR_ARG (-1)        /* NULL / out-of-range argument                  */
#define PFC_ERR_SPECIES (-2)    /* species outside 0..3 or bad sys_offsets       */
#define PFC_ERR_WORKSPACE (-3)  /* workspace missing, misaligned or too small    */
#define PFC_ERR_CUDA (-4)       /* a CUDA runtime call failed                    */
#define PFC_ERR_CAPTURE (-5)    /* graph capture / instantiate failed            */
#define PFC_ERR_STATE (-6)      /* no bound state, or another CUDA device current */

/* sticky device status bits (pfc_status) */
#define PFC_STATUS_RADIAL_OVERFLOW 1u   /* an atom has more radial neighbours than its row holds (min(192, N_sys-1)) */
#define PFC_STATUS_ANGULAR_OVERFLOW 2u  /* reserved (never set: angular neighbours are flagged radial entries) */
#define PFC_STATUS_ANGULAR_ROW 4u       /* one atom has > PFC_MAX_ANGULAR angular neighbours */
#define PFC_STATUS_NONFINITE 8u         /* a system energy is NaN/Inf            */
#define PFC_STATUS_CELL_OVERFLOW 16u    /* cell grid exceeded its capacity       */

#define PFC_AEV_LEN 384                 /* 64 radial + 320 angular (configs[0])  */
#define PFC_N_WEIGHTS 378756            /* 4 elements x 94,689 (O5)    */
#define PFC_MAX_ANGULAR 96              /* angular neighbours one atom may have  */

#define PFC_MLP_FP32 0                  /* FP32 FFMA grouped MLP                 */
#define PFC_MLP_TENSOR 1                /* tcgen05 kind::f16, fp16 hi|lo 3-term split, fp32 accumulate */
#define PFC_MLP_TENSOR_1TERM 2          /* tcgen05 plain fp16 operands: tolerance evidence only (fails it) */
#define PFC_MLP_AUTO 3                  /* TENSOR for batches of >= 1024 atoms if its calibration check passes, FP32 otherwise */

/* Optional tuning knobs, passed explicitly through pfc_desc_t.tuning (HOST pointer, NULL = all
 * defaults; a zero-filled struct is also "all defaults").  The library reads no environment
 * variables.  None of them is needed in production; the tests use them to reach every kernel variant. */
typedef struct {
  int32_t k3_tile_rows;       /* FP32 MLP tile height: 0 = chosen by pfc_create from the batch; 16, 32, 64 or 128 */
  int32_t k3_deep_ring;       /* FP32 MLP weight staging: 0 = chosen by pfc_create; 1 = two buffers;
                                 2 = eight-stage ring (tiles of <= 32 rows only, ignored otherwise) */
  int32_t tc_comp_override;   /* 0 = truncation compensation of the tensor-core MLP calibrated per handle on its first
                                 batch; 1 = no calibration: the two scales below (0 switches
                                 the compensation off) */
  float tc_comp_forward;      /* used when tc_comp_override = 1 */
  float tc_comp_backward;
  int32_t steps_per_graph;    /* MD steps captured per CUDA graph by pfc_step: 0 = default (16); >= 1 */
  int32_t k3_cluster;         /* FP32 MLP of a batch of at most 18 16-row tiles (a single small molecule): 0 = one
                                 cluster of 8 CTAs per tile (unless k3_tile_rows / k3_deep_ring ask for a variant);
                                 1 = never; 2 = required (PFC_ERR_ARG if the batch has more tiles) */
  int32_t skin_list;          /* systems above 2,048 atoms (cell list): 0 = neighbour rows rebuilt from the cell list every
                                 evaluation (default); 1 = candidate rows with a 0.5 A skin, rebuilt only when an atom
                                 has moved more than 0.25 A since the build, the exact predicate applied to the candidates
                                 every evaluation (the lists are the same bit for bit; pays when atoms move slowly) */
} pfc_tuning_t;

typedef struct pfc_ctx pfc_t;           /* opaque; owned by the library          */

/* All pointers in the descriptor are HOST pointers except `workspace`;
 * everything is copied during pfc_create and may be freed afterwards
 * (the workspace must outlive the handle). */
typedef struct {
  int32_t n_atoms;               /* >= 1                                           */
  int32_t n_systems;             /* >= 1                                           */
  const int32_t *species;        /* HOST [n_atoms], 0=H 1=C 2=N 3=O               */
  const int32_t *sys_offsets;    /* HOST [n_systems+1], ascending, [0]=0, last=n_atoms */
  const float *weights;          /* HOST [PFC_N_WEIGHTS]; per element e=0..3:
                                    W1[160][384] b1[160] W2[128][160] b2[128]
                                    W3[96][128] b3[96] W4[1][96] b4[1], row-major [out][in] */
  const float *masses_amu;       /* HOST [4] or NULL -> {1.008,12.011,14.007,15.999} */
  void *workspace;               /* DEVICE, 256-byte aligned, >= pfc_workspace_bytes() */
  size_t workspace_bytes;
  int32_t mlp_path;              /* PFC_MLP_AUTO (recommended), PFC_MLP_FP32, PFC_MLP_TENSOR (or PFC_MLP_TENSOR_1TERM) */
  const pfc_tuning_t *tuning;    /* HOST or NULL (defaults)                         */
} pfc_desc_t;

/* Bytes of device workspace pfc_create needs for these sizes (0 on bad args). */
size_t pfc_workspace_bytes(int32_t n_atoms, int32_t n_systems);

/* Validates the descriptor, builds the static element grouping and the neighbour-row layout,
 * uploads the weights (synchronous copies on the legacy stream) and returns a handle bound to the
 * CUDA device that is current at this call; every later call on the handle must be made with the
 * same device current (PFC_ERR_STATE otherwise). */
int pfc_create(const pfc_desc_t *desc, pfc_t **out);

/* Energy and forces at the given positions (explicit-force
 * return as in PAPER.md:121).  pos: DEVICE [n_atoms] float4 (read only).
 * E: DEVICE [n_systems] floats, potential energy per system.  F: DEVICE
 * [n_atoms] float4 = {-dE/dx, -dE/dy, -dE/dz, e_i}.  stream: a cudaStream_t
 * (NULL = legacy default stream).  Enqueues: neighbour build (K1), AEV (K2),
 * MLP forward/backward (K3), force chain rule + gather (K4), energy sum -- as ONE replay of a
 * CUDA graph captured the first time this (pos, E, F) triple of buffers is seen (the paper's
 * CUDA-Graph finding; the four most recent triples stay cached). */
int pfc_energy_forces(pfc_t *ctx, const float *pos, float *E, float *F, void *stream);

/* The provider call in the paper's own units: the callback of
 * PAPER.md:29-47 receives positions in nm and returns the potential energy in kJ/mol
 * ("RETURN_ENERGY", forces then follow by differentiation) or energy and
 * explicit forces in kJ/mol/nm.  pos_nm DEVICE [n_atoms][3] packed float;
 * E_kj DEVICE [n_systems]; F_kj_nm DEVICE [n_atoms][3] packed float, or NULL for the
 * energy-only mode.  Packing, the whole of pfc_energy_forces and the conversion (1 nm = 10 A,
 * 1 eV = 96.485332 kJ/mol) are enqueued on `stream`; nothing is synchronised.  Uses internal
 * staging buffers: PFC_ERR_STATE if a pfc_run_host state is currently bound to them. */
int pfc_energy_forces_nm(pfc_t *ctx, const float *pos_nm, float *E_kj, float *F_kj_nm, void *stream);

/* Binds (does not copy) the MD state advanced by pfc_step: pos, vel DEVICE
 * [n_atoms] float4, updated in place; E DEVICE [n_systems]; F DEVICE [n_atoms]
 * float4 (forces/energies of the last completed step).  Resets the internal
 * position-compensation words and marks forces as stale so that the next
 * pfc_step evaluates them at the bound positions first. */
int pfc_set_state(pfc_t *ctx, float *pos, float *vel, float *E, float *F, void *stream);

/* n_steps of velocity-Verlet (O8) with time step dt_fs
 * on the bound state, on the bound stream, by replaying one captured CUDA
 * graph per step with no host round trip.  On return (after the caller syncs
 * the stream) pos, vel, F, E hold the synchronous (x_n, v_n, F(x_n), E(x_n)). */
int pfc_step(pfc_t *ctx, int32_t n_steps, float dt_fs);

/* n_steps of Langevin dynamics on the bound state (the paper's timing
 * protocol is a Langevin integrator with friction 0.1 ps^-1; O9, readings
 * S27/S28): BAOAB on the velocity-Verlet kicks,
 *   v += dt/2 a;  x += dt/2 v;  v = c1 v + c2 sqrt(kB T ACC/m) xi;  x += dt/2 v;  forces;  v += dt/2 a,
 * c1 = exp(-friction dt), c2 = sqrt(1 - c1^2).  friction_per_fs in fs^-1 (0.1 ps^-1 = 1e-4),
 * temperature_K in kelvin.  xi are standard normals from Philox4x32-10 with counter
 * (global atom index, step index, 0, 0) and key = seed, Box-Muller in fp32; the step index counts
 * Langevin steps since pfc_set_state, starting at 1, and lives in device memory, so a step is one
 * replayed CUDA graph like pfc_step.  friction 0 reproduces pfc_step up to rounding.
 * Same asynchrony, state and error conventions as pfc_step. */
int pfc_step_langevin(pfc_t *ctx, int32_t n_steps, float dt_fs, float friction_per_fs,
                      float temperature_K, uint64_t seed);

/* Trajectory frames (the paper's protocol writes 10 frames per 1000 steps): binds
 * frames DEVICE [max_frames][n_atoms] float4 (caller-owned; NULL unbinds).  Every later pfc_step /
 * pfc_step_langevin call copies the positions after each stride-th step (counted since
 * pfc_set_state) into the next frame, device to device on the bound stream, until max_frames are
 * written.  pfc_frames_written returns the count (host bookkeeping; sync the stream before reading
 * the frames). */
int pfc_set_frames(pfc_t *ctx, float *frames, int32_t stride, int32_t max_frames);
int pfc_frames_written(pfc_t *ctx, int32_t *n);

/* Host-buffer convenience path (used for end-to-end timing): copies pos/vel
 * HOST [n_atoms][4] to internal device buffers, runs n_steps, copies pos, vel,
 * F (optional, may be NULL) and E HOST [n_systems] back, and synchronises. */
int pfc_run_host(pfc_t *ctx, float *pos_host, float *vel_host, int32_t n_steps, float dt_fs,
                 float *E_host, float *F_host, void *stream);

/* As pfc_run_host, for a caller that keeps the MD state on the host between calls (the callback
 * regime of PAPER.md:29-47: one force evaluation per step): F_host HOST [n_atoms][4] is REQUIRED and
 * on entry holds the forces at pos_host as a previous pfc_run_host / pfc_run_host_resume returned
 * them; they are uploaded instead of being recomputed, so n_steps cost n_steps force evaluations
 * (pfc_run_host costs n_steps + 1).  Passing forces that do not belong to pos_host is undefined. */
int pfc_run_host_resume(pfc_t *ctx, float *pos_host, float *vel_host, float *F_host, int32_t n_steps,
                        float dt_fs, float *E_host, void *stream);

/* Parity getters: DEVICE pointers into the workspace, valid until the next
 * call that enqueues work.  Lists are int32 CSR, rows ascending by neighbour
 * index (O2/S7): the "deterministically ordered pair list" of north_star (1).
 * pfc_get_neighbors enqueues, on the handle's stream, the export of the last evaluation's
 * fixed-capacity rows (the step path's own format) into that CSR; synchronise before reading. */
int pfc_get_neighbors(pfc_t *ctx, const int32_t **r_off, const int32_t **r_idx,
                      const int32_t **a_off, const int32_t **a_idx);
/* aev, g: [n_rows][384] in element-sorted padded row order; row_of_atom
 * DEVICE [n_atoms] gives each atom's row.  (On the tensor-core MLP path K2 writes the AEV as the
 * MLP's packed fp16 hi|lo operand image; the call then enqueues its unpacking into fp32 rows on the
 * handle's stream: synchronise before reading.) */
int pfc_get_intermediates(pfc_t *ctx, const float **aev, const float **g,
                          const int32_t **row_of_atom, int32_t *n_rows);

/* Synchronises the bound/last-used stream and returns the sticky status bits. */
int pfc_status(pfc_t *ctx, uint32_t *bits);

int pfc_destroy(pfc_t *ctx);
const char *pfc_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* PFC_H_ */
