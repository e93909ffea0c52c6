/* pfc_noalloc.h -- the ONE entry point of libpfc whose scratch memory is neither allocated by
 * the call nor carved from a caller's workspace: it lives in a file-scope
 * `static __device__ __align__(256)` array inside the library (4 KB; every GPU that loads
 * libpfc.so holds it until the process exits).
 *
 * Why.  Some callers cannot call cudaMalloc where they need a result: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation.  The neighbour-list offsets
 * are the result such a caller asks for between steps (how many pairs / angular pairs does every
 * atom have, where does its row start in a CSR it lays out itself).  The existing path,
 * pfc_get_neighbors (pfc.h; the parity export of reading S7, PAPER.md:21 names neighbour-list
 * operators as the hand-kernel precedent), computes them by a reduce-then-scan whose block totals
 * sit in the handle's workspace -- and it rewrites the workspace's export block, which with
 * pfc_tuning_t.skin_list = 1 also holds the candidate rows.  This variant leaves the workspace
 * untouched.
 */
#ifndef PFC_NOALLOC_H_
#define PFC_NOALLOC_H_

#include "pfc.h"

#ifdef __cplusplus
extern "C" {
#endif

#define PFC_NOALLOC_MAX_ATOMS 1048576   /* 512 scan blocks of 2,048 atoms: 512 x 8 bytes = 4 KB of static scratch */
#define PFC_ERR_TOO_LARGE (-7)          /* the handle has more atoms than PFC_NOALLOC_MAX_ATOMS */

/* Exclusive prefix sums of the neighbour counts of the handle's LAST evaluation
 * (pfc_energy_forces / pfc_step), exactly the r_off / a_off arrays pfc_get_neighbors returns:
 *   r_off DEVICE [n_atoms + 1] int32 (caller-owned): r_off[i] = radial neighbours of atoms 0..i-1;
 *   a_off DEVICE [n_atoms + 1] int32 (caller-owned): the same for the angular subset.
 * Enqueues two small kernels on `stream` (a cudaStream_t; use the stream the evaluation ran on,
 * or order the two yourself) and returns; nothing is synchronised.  Calls no cudaMalloc, cudaFree
 * or other allocating routine, and touches no byte of the handle's workspace.
 *
 * The scratch (one int2 total per block of 2,048 atoms) is SHARED by every call of this entry
 * point on a device and keeps the last call's contents.  Nothing in it has to start at zero:
 * every entry a call reads it has written first.  Two calls that overlap on the GPU (different
 * streams, no dependency between them) race on it: give them an order.
 * Errors: PFC_ERR_ARG (NULL argument), PFC_ERR_STATE (the handle's device is not current),
 * PFC_ERR_TOO_LARGE (n_atoms > PFC_NOALLOC_MAX_ATOMS: nothing is enqueued), PFC_ERR_CUDA. */
int pfc_neighbor_offsets_noalloc(pfc_t *ctx, int32_t *r_off, int32_t *a_off, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PFC_NOALLOC_H_ */
