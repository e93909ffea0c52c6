// pfc_api.cu -- the C ABI of include/pfc.h: workspace carving, static element
// grouping, weight repacking, kernel sequencing and CUDA-graph capture/replay.
// Device memory and streams come from the caller (PyTorch); the library calls
// no allocator.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <cmath>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/pfc.h"
#include "../../include/pfc_debug.h"
#include "../../include/pfc_noalloc.h"
#include "k0_units.cuh"
#include "k1_neighbors.cuh"
#include "k2_aev.cuh"
#include "k3_mlp_fp32.cuh"
#include "k3_mlp_cluster.cuh"
#include "k3_mlp_tc.cuh"
#include "tc_probe.cuh"
#include "k4_forces.cuh"
#include "k5_verlet.cuh"

using namespace pfc;

namespace {

constexpr size_t ALIGN = 256;
constexpr int CALIB_NSTAT = 6;                // calibration, per 128-row block: sum e^2, sum de e, sum g^2, sum dg g, max|de|, max|dg|
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

// per-element FFMA weight block on the device (floats): packed phase images, then b1 b2 b3 w4 b4
constexpr int DEV_W_PER_ELEM = MLP_P_FLOATS + MLP_V_FLOATS;
static_assert(MLP_P_FLOATS % 4 == 0 && DEV_W_PER_ELEM % 4 == 0, "16-byte aligned blocks");

struct Carver {                 // bump allocator over the caller's workspace (or a dry run)
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <typename T>
  T* take(size_t n) {
    off = align_up(off);
    T* p = base ? (T*)(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

struct Sizes {
  int n_atoms, n_systems, n_rows;
  int cap_r;                                  // neighbour-row entries (sum of the row capacities, worst case)
  int n_items;                                // K1 brute-force work items (worst case)
  size_t rank_words;                          // rank-table words (worst case: every system BRUTE_MAX atoms)
  int n_scan_blocks;
  int n_cell_sys, n_cell_atoms, cell_slots;   // cell_slots: pooled cell arrays (incl. +1 per system)
};

struct Buffers {
  int *species, *sys_off, *row_of_atom;
  float4 *xs, *xsl;
  int4* items;                  // K1 brute-force work items
  int* row_beg;                 // [N+1] first entry of every atom's fixed-capacity neighbour row
  uint32_t* nbr;                // [cap_r] entry words (k1_neighbors.cuh)
  int4* rank_info;              // [N] {first word of the atom's rank table or -1 (cell-list system), first atom of its system, words per atom, 0}
  int2* rank_tab;               // brute-force systems: per atom ceil(N_sys / 32) words {ballot, entries before} (K1 -> K4a)
  int2 *cnt, *block_tot;
  int *r_off, *a_off, *r_idx, *a_idx;   // CSR export (pfc_get_neighbors only); r_idx | a_idx are one block ...
  uint32_t* cand;               // ... which between exports holds the cell-list systems' candidate rows (skin list)
  int* ccnt;                    // [cell atoms] candidates per atom
  float4* x_build;              // [cell atoms] positions at the last candidate build
  int* skin_state;              // [4] {rebuild flag, builds so far}
  float *aev, *g, *e_row;       // aev: fp32 rows (FP32 MLP) or the packed fp16 operand image (tensor MLP), same bytes
  float* aev_unpacked;          // pfc_get_intermediates on the tensor path; calibration: fp32 AEV rows, then the FP32 MLP's g
  float* e_ref;                 // calibration: the FP32 MLP's per-row energies
  double* calib_part;           // calibration: per 128-row block partial sums
  float4 *edge, *self, *xlo;
  uint32_t* status;
  StepParams* sp;
  unsigned long long* work;     // pfc_work_counts
  long long* trace;             // pfc_k3_timeline
  float* weights;
  float* wcl;                   // cluster MLP (single small molecule): per element and cluster rank, the six weight slices
  uint8_t* wtc;                 // tensor-core path: packed hi|lo swizzled weight chunks
  float* bias_tc;
  // cell list
  int *cell_sys, *cell_cap_base, *cell_slot_base, *cell_atom_list, *atom_cell_sys, *atom_cell;
  int *cell_count, *cell_start, *cell_cursor;
  float4* cell_xyz;             // positions in cell order, atom index | species << 29 in .w
  CellGrid* grids;
  // internal state for pfc_run_host / pfc_energy_forces_nm
  float4 *h_pos, *h_vel, *h_frc;
  float* h_E;
};

size_t carve(const Sizes& s, void* base, Buffers* b) {
  Carver c(base);
  Buffers t;
  const size_t N = (size_t)s.n_atoms;
  t.species = c.take<int>(N);
  t.sys_off = c.take<int>((size_t)s.n_systems + 1);
  t.row_of_atom = c.take<int>(N);
  t.xs = c.take<float4>(N);
  t.xsl = c.take<float4>(N);
  t.items = c.take<int4>((size_t)s.n_items);
  t.row_beg = c.take<int>(N + 1);
  t.nbr = c.take<uint32_t>((size_t)s.cap_r);
  t.rank_info = c.take<int4>(N);
  t.rank_tab = c.take<int2>(s.rank_words + 1);
  t.cnt = c.take<int2>(N);
  t.block_tot = c.take<int2>((size_t)s.n_scan_blocks);
  t.r_off = c.take<int>(N + 1);
  t.a_off = c.take<int>(N + 1);
  t.r_idx = c.take<int>(2 * (size_t)s.cap_r);             // r_idx | a_idx contiguous: 2 x 192 = CAND_CAP words per cell-list atom
  t.a_idx = t.r_idx ? t.r_idx + s.cap_r : nullptr;
  t.cand = (uint32_t*)t.r_idx;
  t.aev = c.take<float>((size_t)s.n_rows * AEV_LEN);
  t.g = c.take<float>((size_t)s.n_rows * AEV_LEN);
  t.aev_unpacked = c.take<float>((size_t)s.n_rows * AEV_LEN);
  t.e_row = c.take<float>((size_t)s.n_rows);
  t.e_ref = c.take<float>((size_t)s.n_rows);
  t.calib_part = c.take<double>((size_t)(s.n_rows / ROW_PAD) * CALIB_NSTAT);
  t.edge = c.take<float4>((size_t)s.cap_r);
  t.self = c.take<float4>(N);
  t.xlo = c.take<float4>(N);
  t.status = c.take<uint32_t>(64);
  t.sp = c.take<StepParams>(1);
  t.work = c.take<unsigned long long>(8);
  t.trace = c.take<long long>((size_t)TC_TRACE_STRIDE * TC_TRACE_ITERS);
  t.weights = c.take<float>((size_t)NSPEC * DEV_W_PER_ELEM);
  t.wcl = c.take<float>((size_t)NSPEC * CL_SIZE * CL_W_FLOATS);
  t.wtc = c.take<uint8_t>((size_t)NSPEC * TC_W_BYTES_PER_ELEM);
  t.bias_tc = c.take<float>((size_t)NSPEC * TC_BIAS_LEN);
  t.cell_sys = c.take<int>((size_t)s.n_cell_sys + 1);
  t.cell_cap_base = c.take<int>((size_t)s.n_cell_sys + 1);
  t.cell_slot_base = c.take<int>((size_t)s.n_cell_sys + 1);
  t.grids = c.take<CellGrid>((size_t)s.n_cell_sys + 1);
  t.cell_atom_list = c.take<int>((size_t)s.n_cell_atoms + 1);
  t.atom_cell_sys = c.take<int>((size_t)s.n_cell_atoms + 1);
  t.atom_cell = c.take<int>((size_t)s.n_cell_atoms + 1);
  t.cell_xyz = c.take<float4>((size_t)s.n_cell_atoms + 1);
  t.x_build = c.take<float4>((size_t)s.n_cell_atoms + 1);
  t.ccnt = c.take<int>((size_t)s.n_cell_atoms + 1);
  t.skin_state = c.take<int>(4);
  t.cell_count = c.take<int>((size_t)s.cell_slots + 1);
  t.cell_start = c.take<int>((size_t)s.cell_slots + 1);
  t.cell_cursor = c.take<int>((size_t)s.cell_slots + 1);
  t.h_pos = c.take<float4>(N);
  t.h_vel = c.take<float4>(N);
  t.h_frc = c.take<float4>(N);
  t.h_E = c.take<float>((size_t)s.n_systems);
  if (b) *b = t;
  return align_up(c.off);
}

inline int cells_for(int n_sys_atoms) { return n_sys_atoms + 64 + 1; }
// default scale of the tensor-core MLP's truncation compensation, forward / backward phases
constexpr float TC_LAMBDA_FWD = 0.85f, TC_LAMBDA_BWD = 0.85f;   // uncalibrated elements (fewer than CALIB_MIN_ROWS atoms)
constexpr int CALIB_MIN_ROWS = 256;           // atoms of an element below which its lambdas stay at the defaults
// a calibrated element keeps the tensor path only if, against the FP32 MLP on the same batch, the least-squares
// slopes of its e_i and g errors and its largest errors (relative to the rms of e_i / g) stay below these
// (the slope of e_i is a weak statistic when the e_i of an element are nearly equal -- 500 O atoms of a water
// cluster: it then measures an offset of 1e-7 eV, not a scale -- so its bound sits 5x inside the 1e-5 energy bar
// instead of at the level of the g slope, which is what a trajectory feels)
constexpr double CALIB_MAX_SLOPE_E = 2e-6, CALIB_MAX_SLOPE_G = 3e-7, CALIB_MAX_DE = 1e-4, CALIB_MAX_DG = 5e-5;
// PFC_MLP_AUTO: the tensor-core MLP from this many atoms on.  Its cost is one tile chain (33 us) until the
// batch has more tiles than SMs; measured ms/step, FP32 / tensor (round 2): 1,100 atoms 0.062 / 0.049, 2,200 atoms
// 0.091 / 0.051, config 2 (1,500) 0.081 / 0.069, config 1 (5,632) 0.139 / 0.061.  Below, the FP32 kernels (the
// cluster kernel up to 18 16-row tiles, 15 us)
constexpr int TC_AUTO_MIN_ATOMS = 1024;
constexpr int ROW_CAP = 192;                  // neighbour-row capacity of an atom: min(ROW_CAP, N_sys - 1); bulk at 0.1 / A^3 has 59
constexpr int K1_MIN_BLOCK = 8, K1_MAX_BLOCK = 64;   // atoms per K1 brute-force work item

// worst case over all species / system layouts with these totals
Sizes worst_case_sizes(int n_atoms, int n_systems) {
  Sizes s{};
  s.n_atoms = n_atoms; s.n_systems = n_systems;
  s.n_rows = (n_atoms + ROW_PAD - 1) / ROW_PAD * ROW_PAD + NSPEC * ROW_PAD;
  long long per_r = n_atoms - 1 < ROW_CAP ? n_atoms - 1 : ROW_CAP;      // one system holding every atom
  long long cr = (long long)n_atoms * (per_r > 1 ? per_r : 1);
  s.cap_r = (int)(cr > 2000000000LL ? 2000000000LL : cr);
  s.n_items = n_atoms / K1_MIN_BLOCK + n_systems + 1;
  s.rank_words = (size_t)n_atoms * (size_t)(((n_atoms < BRUTE_MAX ? n_atoms : BRUTE_MAX) + 31) / 32);
  s.n_scan_blocks = (n_atoms + SCAN_BLOCK - 1) / SCAN_BLOCK;
  s.n_cell_sys = n_atoms / (BRUTE_MAX + 1) + 1;
  if (s.n_cell_sys > n_systems) s.n_cell_sys = n_systems;
  s.n_cell_atoms = n_atoms;
  s.cell_slots = n_atoms + 65 * s.n_cell_sys;
  return s;
}

}  // namespace

constexpr int EF_CACHE = 4;                    // pfc_energy_forces graphs kept (most recently used buffer triples)

struct EfGraph {                               // one captured force evaluation: K1 .. energy sum
  const float4* pos = nullptr;
  float* E = nullptr;
  float4* F = nullptr;
  bool with_xlo = false;                       // captured with the bound state's low position words
  cudaGraphExec_t exec = nullptr;
  unsigned long long last_use = 0;
};

struct pfc_ctx {
  Sizes sz;
  Buffers b;
  MlpParams mlp;
  ClParams clp;
  bool skin_list = false;       // cell-list systems: candidate rows with a skin, reused between rebuilds (pfc_tuning_t.skin_list)
  bool mlp_cluster = false;     // FP32 MLP of a batch of <= CL_MAX_TILES 16-row tiles: one cluster of 8 CTAs per tile
  TcParams tcp;
  int device = 0;               // the CUDA device the handle was created on
  int mlp_path;
  int mlp_requested = PFC_MLP_AUTO;
  // tensor-core MLP: truncation compensation
  std::vector<float> bias_host;               // host copy of the per-element tables (ks / kb are rewritten)
  int tc_inv_scale[NSPEC][6] = {};
  int tc_terms = 3;
  int count[NSPEC] = {0, 0, 0, 0};
  bool tc_calibrated = false;                 // lambdas final (calibrated, or fixed by pfc_tuning_t)
  float tc_lambda[NSPEC][2];                  // forward / backward
  float tc_resid[NSPEC][4] = {};              // after calibration: slope e, slope g, max|de|/rms e, max|dg|/rms g
  int tc_fallback = 0;                        // 1: AUTO went back to the FP32 MLP because an element failed the check
  int mlp_tm = 128;             // FFMA K3 tile height
  bool mlp_deep = false;        // FFMA K3 staging: 8-stage mbarrier ring (few tiles per SM) or two buffers
  int n_sms = 148;
  int n_cell_sys, n_cell_atoms;
  int n_items = 0;              // K1 brute-force work items
  size_t k1_smem = 0;           // bytes: positions of the largest brute-force system
  long long brute_tests = 0;    // distance tests per evaluation (work counts)
  int launches_ef, launches_step;
  int steps_per_graph = 16;
  // bound MD state
  float4 *pos = nullptr, *vel = nullptr, *frc = nullptr;
  float* E = nullptr;
  cudaStream_t stream = nullptr, cap_stream = nullptr;
  // pfc_run_host*: the new positions go back to the host on a side stream while the forces are evaluated
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_drift = nullptr, ev_copied = nullptr;
  float4* early_pos_dst = nullptr;   // HOST destination of that copy for the step being enqueued, or NULL
  bool bound = false, forces_stale = true;
  float cur_dt = -1.0f;
  // graphs of the bound state: forces; one Verlet / Langevin step; steps_per_graph of them
  cudaGraphExec_t g_forces = nullptr, g_step = nullptr, g_lstep = nullptr, g_stepk = nullptr, g_lstepk = nullptr;
  EfGraph ef[EF_CACHE];         // pfc_energy_forces: graphs keyed on the caller's buffers
  unsigned long long ef_clock = 0;
  float4* frames = nullptr;     // caller's frame buffer (pfc_set_frames)
  int frame_stride = 0, frame_cap = 0, frames_written = 0;
  long long steps_total = 0;    // steps since pfc_set_state (frame cadence)
  float lg_gamma = -1.f, lg_T = -1.f, lg_dt = -1.f;
  unsigned long long lg_seed = 0;
  int launch_counter = 0;
};

namespace {

#define LAUNCH(ctx, kernel, grid, block, smem, stream, ...)     \
  do {                                                          \
    kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__); \
    ++(ctx)->launch_counter;                                    \
  } while (0)

inline int cdiv(int a, int b) { return (a + b - 1) / b; }

inline bool on_device(const pfc_ctx* c) {      // every call must run with the handle's device current
  int dev = -1;
  return cudaGetDevice(&dev) == cudaSuccess && dev == c->device;
}

// K1: neighbour rows of `pos` (and the packed position copies every later kernel reads)
void enqueue_k1(pfc_ctx* c, const float4* pos, bool with_xlo, cudaStream_t st) {
  const Buffers& b = c->b;
  // the low position words belong to the bound MD state only
  const float4* xlo = with_xlo ? b.xlo : nullptr;
  if (c->n_items > 0)
    LAUNCH(c, k1_brute_kernel, c->n_items, K1_WARPS * 32, c->k1_smem, st, b.items, pos, b.species, xlo, b.xs, b.xsl,
           b.row_beg, b.nbr, b.cnt, b.rank_info, b.rank_tab, b.status);
  if (c->n_cell_sys > 0) {
    const int nca = c->n_cell_atoms;
    // skin list on: has any atom moved more than SKIN/2 since the candidate rows were built?  If so the five
    // build kernels run (they return at once otherwise); then the exact predicate on the candidates, every time.
    // Off (the default): the build kernels see a flag that is always set and write the rows themselves.
    const int* flag = c->skin_list ? b.skin_state : b.skin_state + SKIN_ALWAYS;
    if (c->skin_list)
      LAUNCH(c, k1_skin_check_kernel, cdiv(nca, 256), 256, 0, st, nca, b.cell_atom_list, pos, b.x_build, b.skin_state);
    LAUNCH(c, k1_cell_grid_kernel, c->n_cell_sys, CELL_THREADS, 0, st, flag, b.cell_sys, b.sys_off, b.cell_cap_base,
           pos, b.grids, b.cell_count, b.status, c->skin_list ? CELL_EDGE_MIN_SKIN : CELL_EDGE_MIN);
    LAUNCH(c, k1_cell_assign_kernel, cdiv(nca, 256), 256, 0, st, flag, nca, b.cell_atom_list, b.atom_cell_sys, pos,
           b.grids, b.atom_cell, b.cell_count);
    LAUNCH(c, k1_cell_scan_kernel, c->n_cell_sys, CELL_THREADS, 0, st, flag, b.cell_sys, b.cell_slot_base, b.grids,
           b.cell_count, b.cell_start, b.cell_cursor);
    LAUNCH(c, k1_cell_fill_kernel, cdiv(nca, 256), 256, 0, st, flag, nca, b.cell_atom_list, b.atom_cell,
           pos, b.species, b.cell_cursor, b.cell_xyz);
    if (c->skin_list) {
      LAUNCH(c, k1_cell_cand_kernel, cdiv(nca, K1_WARPS), K1_WARPS * 32, 0, st, b.skin_state, nca, b.cell_atom_list,
             b.atom_cell_sys, b.atom_cell, pos, b.grids, b.cell_start, b.cell_xyz, b.cand, b.ccnt, b.x_build, b.status);
      LAUNCH(c, k1_skin_refresh_kernel, cdiv(nca, K1_WARPS), K1_WARPS * 32, 0, st, b.skin_state, nca, b.cell_atom_list,
             pos, b.species, xlo, b.cand, b.ccnt, b.xs, b.xsl, b.row_beg, b.nbr, b.cnt, b.status);
    } else {
      LAUNCH(c, k1_cell_rows_kernel, cdiv(nca, K1_WARPS), K1_WARPS * 32, 0, st, nca, b.cell_atom_list,
             b.atom_cell_sys, b.atom_cell, pos, b.species, xlo, b.grids, b.cell_start, b.cell_xyz, b.xs, b.xsl,
             b.row_beg, b.nbr, b.cnt, b.status);
    }
  }
}

// K2 into `aev`: fp32 rows (PACK16 false) or the tensor MLP's first operand image
void enqueue_k2(pfc_ctx* c, bool pack16, float* aev, cudaStream_t st) {
  const Buffers& b = c->b;
  const int N = c->sz.n_atoms;
  if (!pack16)
    LAUNCH(c, k2_aev_fwd_kernel<false>, cdiv(N, AEV_WARPS), AEV_WARPS * 32, 0, st, N, b.xs, b.xsl, b.row_beg, b.nbr, b.cnt,
           b.row_of_atom, aev, b.status);
  else                                                    // the tensor MLP's first operand, as it sits in shared memory
    LAUNCH(c, k2_aev_fwd_kernel<true>, cdiv(N, AEV_WARPS), AEV_WARPS * 32, 0, st, N, b.xs, b.xsl, b.row_beg, b.nbr, b.cnt,
           b.row_of_atom, aev, b.status);
}

// K3, FP32 FFMA: tile height and staging chosen by pfc_create.  `g` may be `aev` (a tile's AEV rows are
// consumed in its first phase, long before its g rows are written)
void enqueue_k3_fp32(pfc_ctx* c, const float* aev, float* g, float* e_row, cudaStream_t st) {
  const Sizes& s = c->sz;
  if (c->mlp_cluster) {
    LAUNCH(c, k3_mlp_cluster_kernel, c->clp.n_tiles * CL_SIZE, CL_THREADS, CL_SMEM_BYTES, st, c->clp, aev, g, e_row);
    return;
  }
#define K3_LAUNCH(TM_, DEEP_)                                                                          \
  LAUNCH(c, (k3_mlp_fp32_kernel<TM_, DEEP_>), s.n_rows / TM_, (MlpCfg<TM_, DEEP_>::THREADS),             \
         (MlpCfg<TM_, DEEP_>::SMEM), st, c->mlp, aev, g, e_row)
  if (c->mlp_deep) {
    if (c->mlp_tm == 32) K3_LAUNCH(32, true); else K3_LAUNCH(16, true);
  } else {
    switch (c->mlp_tm) {
      case 128: K3_LAUNCH(128, false); break;
      case 64:  K3_LAUNCH(64, false); break;
      case 32:  K3_LAUNCH(32, false); break;
      default:  K3_LAUNCH(16, false); break;
    }
  }
#undef K3_LAUNCH
}

// K3, tcgen05: persistent, one CTA per SM
void enqueue_k3_tc(pfc_ctx* c, cudaStream_t st) {
  const Buffers& b = c->b;
  const int grid = c->tcp.n_tiles < c->n_sms ? c->tcp.n_tiles : c->n_sms;
  if (c->tc_terms == 3)
    LAUNCH(c, k3_mlp_tc_kernel<3>, grid, TC_THREADS, TC_SMEM_BYTES, st, c->tcp, (const uint8_t*)b.aev, b.g, b.e_row);
  else
    LAUNCH(c, k3_mlp_tc_kernel<1>, grid, TC_THREADS, TC_SMEM_BYTES, st, c->tcp, (const uint8_t*)b.aev, b.g, b.e_row);
}

// K1..K4 + energy sum on `st`
// `ev` (optional): events recorded at the seven stage boundaries K1|K2|K3|K4a|K4b|E-sum|
void enqueue_energy_sum(pfc_ctx* c, const float4* F, float* E, cudaStream_t st) {
  const Buffers& b = c->b;
  if (c->n_cell_sys > 0) LAUNCH(c, k_energy_sum_kernel<1024>, c->sz.n_systems, 1024, 0, st, b.sys_off, F, E, b.status);
  else LAUNCH(c, k_energy_sum_kernel<128>, c->sz.n_systems, 128, 0, st, b.sys_off, F, E, b.status);
}

// `with_esum` false: the per-system energies are not formed (the steps inside a pfc_step call: nobody can read E
// between them; run_steps sums once at the end)
void enqueue_forces(pfc_ctx* c, const float4* pos, float* E, float4* F, bool with_xlo, cudaStream_t st,
                    cudaEvent_t* ev = nullptr, bool with_esum = true) {
  auto mark = [&](int k) { if (ev) cudaEventRecord(ev[k], st); };
  mark(0);
  const Sizes& s = c->sz;
  const Buffers& b = c->b;
  const int N = s.n_atoms;
  enqueue_k1(c, pos, with_xlo, st);
  mark(1);
  enqueue_k2(c, c->mlp_path != PFC_MLP_FP32, b.aev, st);
  mark(2);
  if (c->mlp_path == PFC_MLP_FP32) enqueue_k3_fp32(c, b.aev, b.g, b.e_row, st);
  else enqueue_k3_tc(c, st);
  mark(3);
  LAUNCH(c, k4a_aev_bwd_kernel, cdiv(N, AEV_WARPS), AEV_WARPS * 32, 0, st, N, b.xs, b.xsl, b.row_beg, b.nbr, b.cnt,
         b.row_of_atom, b.rank_info, b.rank_tab, b.g, b.edge, b.self);
  mark(4);
  LAUNCH(c, k4b_gather_kernel, cdiv(N, K4B_ATOMS), K4B_WARPS * 32, 0, st, N, b.row_beg, b.nbr, b.cnt, b.rank_info, b.edge,
         b.self, b.row_of_atom, b.e_row, F);
  mark(5);
  if (with_esum) enqueue_energy_sum(c, F, E, st);
  mark(6);
}

// ---- truncation compensation of the tensor-core MLP ----------------------
// ks[q] = 2^-(operand scales of epilogue q), kb[q] = beta_q ks[q], beta_q = lambda n_q 2.15e-8 with n_q the
// MMA instructions of the accumulator chain and lambda = tc_lambda[e][q < 3 ? 0 : 1]
int upload_tc_factors(pfc_ctx* c, cudaStream_t st) {
  for (int e = 0; e < NSPEC; ++e) {
    float* bt = c->bias_host.data() + (size_t)e * TC_BIAS_LEN;
    for (int q = 0; q < 6; ++q) {
      const float beta = c->tc_lambda[e][q < 3 ? 0 : 1] * (float)tc_chain_mmas(q, c->tc_terms) * 2.15e-8f;
      bt[TC_BIAS_KS + q] = ldexpf(1.0f, c->tc_inv_scale[e][q]);
      bt[TC_BIAS_KB + q] = ldexpf(beta, c->tc_inv_scale[e][q]);
    }
    if (cudaMemcpyAsync(c->b.bias_tc + (size_t)e * TC_BIAS_LEN + TC_BIAS_KS, bt + TC_BIAS_KS, sizeof(float) * 12,
                        cudaMemcpyHostToDevice, st) != cudaSuccess)
      return PFC_ERR_CUDA;
  }
  return PFC_OK;
}

// per 128-row block (one element): sums over its real rows of the FP32 MLP's outputs (ref) and the
// differences of the tensor MLP's outputs to them; fixed order, one owner per partial
__global__ void __launch_bounds__(256)
k_calib_stats_kernel(const __grid_constant__ MlpParams P, const float* __restrict__ g_ref, const float* __restrict__ g_tc,
                     const float* __restrict__ e_ref, const float* __restrict__ e_tc, double* __restrict__ part) {
  __shared__ double sh[8][CALIB_NSTAT];
  const int row0 = blockIdx.x * ROW_PAD, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int el = 0;
#pragma unroll
  for (int k = 1; k < NSPEC; ++k) el += (row0 >= P.row_start[k]);
  const int rend = min(row0 + ROW_PAD, P.row_end[el]);
  double see = 0.0, sde = 0.0, sgg = 0.0, sdg = 0.0, mde = 0.0, mdg = 0.0;
  for (int r = row0 + warp; r < rend; r += 8) {
    for (int col = lane; col < AEV_LEN; col += 32) {
      const float a = g_ref[(size_t)r * AEV_LEN + col], d = g_tc[(size_t)r * AEV_LEN + col] - a;
      sgg += (double)a * a; sdg += (double)d * a; mdg = fmax(mdg, (double)fabsf(d));
    }
    if (lane == 0) {
      const float a = e_ref[r], d = e_tc[r] - a;
      see += (double)a * a; sde += (double)d * a; mde = fmax(mde, (double)fabsf(d));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    see += __shfl_xor_sync(0xffffffffu, see, o); sde += __shfl_xor_sync(0xffffffffu, sde, o);
    sgg += __shfl_xor_sync(0xffffffffu, sgg, o); sdg += __shfl_xor_sync(0xffffffffu, sdg, o);
    mde = fmax(mde, __shfl_xor_sync(0xffffffffu, mde, o)); mdg = fmax(mdg, __shfl_xor_sync(0xffffffffu, mdg, o));
  }
  if (lane == 0) { sh[warp][0] = see; sh[warp][1] = sde; sh[warp][2] = sgg; sh[warp][3] = sdg; sh[warp][4] = mde; sh[warp][5] = mdg; }
  __syncthreads();
  if (threadIdx.x < CALIB_NSTAT) {
    double v = sh[0][threadIdx.x];
    for (int w = 1; w < 8; ++w) v = threadIdx.x < 4 ? v + sh[w][threadIdx.x] : fmax(v, sh[w][threadIdx.x]);
    part[(size_t)blockIdx.x * CALIB_NSTAT + threadIdx.x] = v;
  }
}

// Calibrates the two compensation scales of every element on the batch at `pos` against the
// library's own FP32 MLP (never the oracle): K1, K2 (fp32 rows), FP32 MLP -> reference e_i, g; K2 (operand
// image), then the tensor MLP with (lambda_f, lambda_b) = (0,0), (1,0), (0,1): the error slopes are linear in
// both, solved per element; one more run checks the result.  With PFC_MLP_AUTO an element that misses the
// check sends the whole handle back to the FP32 MLP.  Synchronises `st` (first use of a handle only).
int calibrate_tc(pfc_ctx* c, const float4* pos, bool with_xlo, cudaStream_t st) {
  const Buffers& b = c->b;
  const int n_blocks = c->sz.n_rows / ROW_PAD;
  enqueue_k1(c, pos, with_xlo, st);
  enqueue_k2(c, false, b.aev_unpacked, st);
  enqueue_k3_fp32(c, b.aev_unpacked, b.aev_unpacked, b.e_ref, st);
  enqueue_k2(c, true, b.aev, st);
  std::vector<double> part((size_t)n_blocks * CALIB_NSTAT);
  struct Stat { double see = 0, sde = 0, sgg = 0, sdg = 0, mde = 0, mdg = 0; };
  auto run = [&](Stat* out) -> int {
    int rc = upload_tc_factors(c, st);
    if (rc != PFC_OK) return rc;
    enqueue_k3_tc(c, st);
    LAUNCH(c, k_calib_stats_kernel, n_blocks, 256, 0, st, c->mlp, b.aev_unpacked, b.g, b.e_ref, b.e_row, b.calib_part);
    if (cudaMemcpyAsync(part.data(), b.calib_part, sizeof(double) * part.size(), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
      return PFC_ERR_CUDA;
    for (int e = 0; e < NSPEC; ++e) {
      Stat t;
      for (int blk = c->mlp.row_start[e] / ROW_PAD; blk < c->mlp.row_start[e + 1] / ROW_PAD; ++blk) {   // fixed order
        const double* p = part.data() + (size_t)blk * CALIB_NSTAT;
        t.see += p[0]; t.sde += p[1]; t.sgg += p[2]; t.sdg += p[3];
        t.mde = p[4] > t.mde ? p[4] : t.mde; t.mdg = p[5] > t.mdg ? p[5] : t.mdg;
      }
      out[e] = t;
    }
    return PFC_OK;
  };
  auto set_all = [&](float lf, float lb) {
    for (int e = 0; e < NSPEC; ++e)
      if (c->count[e] >= CALIB_MIN_ROWS) { c->tc_lambda[e][0] = lf; c->tc_lambda[e][1] = lb; }
  };
  Stat s00[NSPEC], s10[NSPEC], s01[NSPEC], fin[NSPEC];
  int rc;
  set_all(0.f, 0.f); if ((rc = run(s00)) != PFC_OK) return rc;
  set_all(1.f, 0.f); if ((rc = run(s10)) != PFC_OK) return rc;
  set_all(0.f, 1.f); if ((rc = run(s01)) != PFC_OK) return rc;
  auto slope = [](double sd, double ss) { return ss > 0.0 ? sd / ss : 0.0; };
  auto clamp = [](double v) { return !(v >= 0.0) ? 0.0 : v > 2.5 ? 2.5 : v; };
  for (int e = 0; e < NSPEC; ++e) {
    if (c->count[e] < CALIB_MIN_ROWS) continue;
    const double e0 = slope(s00[e].sde, s00[e].see), e1 = slope(s10[e].sde, s10[e].see);
    const double g0 = slope(s00[e].sdg, s00[e].sgg), g1 = slope(s10[e].sdg, s10[e].sgg), g2 = slope(s01[e].sdg, s01[e].sgg);
    const double lf = fabs(e1 - e0) > 1e-9 ? clamp(-e0 / (e1 - e0)) : TC_LAMBDA_FWD;
    const double lb = fabs(g2 - g0) > 1e-9 ? clamp(-(g0 + (g1 - g0) * lf) / (g2 - g0)) : TC_LAMBDA_BWD;
    c->tc_lambda[e][0] = (float)lf; c->tc_lambda[e][1] = (float)lb;
  }
  if ((rc = run(fin)) != PFC_OK) return rc;
  bool ok = true;
  for (int e = 0; e < NSPEC; ++e) {
    if (c->count[e] < CALIB_MIN_ROWS) continue;
    const double n = (double)c->count[e];
    const double rms_e = sqrt(fin[e].see / n), rms_g = sqrt(fin[e].sgg / (n * AEV_LEN));
    c->tc_resid[e][0] = (float)slope(fin[e].sde, fin[e].see);
    c->tc_resid[e][1] = (float)slope(fin[e].sdg, fin[e].sgg);
    c->tc_resid[e][2] = (float)(rms_e > 0.0 ? fin[e].mde / rms_e : 0.0);
    c->tc_resid[e][3] = (float)(rms_g > 0.0 ? fin[e].mdg / rms_g : 0.0);
    if (!(fabs(c->tc_resid[e][0]) <= CALIB_MAX_SLOPE_E) || !(fabs(c->tc_resid[e][1]) <= CALIB_MAX_SLOPE_G) ||
        !(c->tc_resid[e][2] <= CALIB_MAX_DE) || !(c->tc_resid[e][3] <= CALIB_MAX_DG))
      ok = false;
  }
  c->tc_calibrated = true;
  if (!ok && c->mlp_requested == PFC_MLP_AUTO) {          // this weight set / batch is not for the tensor path
    c->mlp_path = PFC_MLP_FP32;
    c->tc_fallback = 1;
  }
  return PFC_OK;
}

inline int ensure_calibrated(pfc_ctx* c, const float4* pos, bool with_xlo, cudaStream_t st) {
  if (c->mlp_path == PFC_MLP_FP32 || c->tc_calibrated) return PFC_OK;
  return calibrate_tc(c, pos, with_xlo, st);
}

template <int MODE>
void enqueue_verlet(pfc_ctx* c, cudaStream_t st) {
  LAUNCH(c, k5_verlet_kernel<MODE>, cdiv(c->sz.n_atoms, K5_THREADS), K5_THREADS, 0, st, c->sz.n_atoms, c->b.sp,
         c->b.species, c->frc, c->pos, c->vel, c->b.xlo);
}

template <int MODE>
void enqueue_langevin(pfc_ctx* c, cudaStream_t st) {
  LAUNCH(c, k5_langevin_kernel<MODE>, cdiv(c->sz.n_atoms, K5_THREADS), K5_THREADS, 0, st, c->sz.n_atoms, c->b.sp,
         c->b.species, c->frc, c->pos, c->vel, c->b.xlo);
}

void drop_state_graphs(pfc_ctx* c) {
  cudaGraphExec_t* gs[] = {&c->g_forces, &c->g_step, &c->g_lstep, &c->g_stepk, &c->g_lstepk};
  for (cudaGraphExec_t* g : gs) {
    if (*g) cudaGraphExecDestroy(*g);
    *g = nullptr;
  }
}

// Captures `n_rep` repetitions of {optional fused integrator kernel, forces} on the private capture
// stream (the caller's may be the legacy stream, which cannot capture); the instantiated graph is
// launched on the caller's stream.  kind 0: forces only; 1: fused Verlet kernel + forces;
// 2: fused Langevin kernel + forces.
int capture(pfc_ctx* c, int kind, int n_rep, const float4* pos, float* E, float4* F, bool with_xlo,
            cudaGraphExec_t* out) {
  cudaGraph_t graph = nullptr;
  if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess)
    return PFC_ERR_CAPTURE;
  if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) return PFC_ERR_CAPTURE;
  for (int r = 0; r < n_rep; ++r) {
    if (kind == 1) enqueue_verlet<2>(c, c->cap_stream);
    if (kind == 2) enqueue_langevin<2>(c, c->cap_stream);
    enqueue_forces(c, pos, E, F, with_xlo, c->cap_stream, nullptr, kind == 0);
  }
  cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
  if (e != cudaSuccess || !graph) { cudaGetLastError(); return PFC_ERR_CAPTURE; }
  e = cudaGraphInstantiate(out, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) { cudaGetLastError(); return PFC_ERR_CAPTURE; }
  return PFC_OK;
}

}  // namespace

extern "C" {

size_t pfc_workspace_bytes(int32_t n_atoms, int32_t n_systems) {
  if (n_atoms < 1 || n_systems < 1 || n_systems > n_atoms) return 0;
  Sizes s = worst_case_sizes(n_atoms, n_systems);
  return carve(s, nullptr, nullptr);
}

int pfc_create(const pfc_desc_t* d, pfc_t** out) {
  if (!d || !out || !d->species || !d->sys_offsets || !d->weights) return PFC_ERR_ARG;
  if (d->n_atoms < 1 || d->n_systems < 1 || d->n_systems > d->n_atoms) return PFC_ERR_ARG;
  if (d->mlp_path != PFC_MLP_FP32 && d->mlp_path != PFC_MLP_TENSOR && d->mlp_path != PFC_MLP_TENSOR_1TERM &&
      d->mlp_path != PFC_MLP_AUTO)
    return PFC_ERR_ARG;
  const int N = d->n_atoms, NS = d->n_systems;
  if (d->sys_offsets[0] != 0 || d->sys_offsets[NS] != N) return PFC_ERR_SPECIES;
  for (int s = 0; s < NS; ++s)
    if (d->sys_offsets[s + 1] <= d->sys_offsets[s]) return PFC_ERR_SPECIES;
  int count[NSPEC] = {0, 0, 0, 0};
  for (int i = 0; i < N; ++i) {
    if (d->species[i] < 0 || d->species[i] >= NSPEC) return PFC_ERR_SPECIES;
    ++count[d->species[i]];
  }
  if (!d->workspace || ((uintptr_t)d->workspace % ALIGN) != 0) return PFC_ERR_WORKSPACE;
  if (d->workspace_bytes < pfc_workspace_bytes(N, NS)) return PFC_ERR_WORKSPACE;

  pfc_tuning_t tun{};                                   // zero = every default
  if (d->tuning) tun = *d->tuning;
  if (tun.k3_tile_rows != 0 && tun.k3_tile_rows != 16 && tun.k3_tile_rows != 32 && tun.k3_tile_rows != 64 &&
      tun.k3_tile_rows != 128)
    return PFC_ERR_ARG;
  if (tun.k3_deep_ring < 0 || tun.k3_deep_ring > 2 || tun.steps_per_graph < 0 || tun.steps_per_graph > 256 ||
      tun.k3_cluster < 0 || tun.k3_cluster > 2 || tun.skin_list < 0 || tun.skin_list > 1)
    return PFC_ERR_ARG;

  pfc_ctx* c = new (std::nothrow) pfc_ctx();
  if (!c) return PFC_ERR_ARG;
  if (cudaGetDevice(&c->device) != cudaSuccess) { cudaGetLastError(); delete c; return PFC_ERR_CUDA; }
  if (tun.steps_per_graph > 0) c->steps_per_graph = tun.steps_per_graph;
  c->skin_list = tun.skin_list == 1;
  c->mlp_requested = d->mlp_path;
  c->mlp_path = d->mlp_path == PFC_MLP_AUTO ? (d->n_atoms >= TC_AUTO_MIN_ATOMS ? PFC_MLP_TENSOR : PFC_MLP_FP32) : d->mlp_path;
  for (int e = 0; e < NSPEC; ++e) c->count[e] = count[e];
  c->sz = worst_case_sizes(N, NS);                      // capacities are the worst-case ones
  // static element grouping: rows sorted by element, blocks padded to ROW_PAD
  int row_start[NSPEC + 1];
  row_start[0] = 0;
  for (int e = 0; e < NSPEC; ++e) row_start[e + 1] = row_start[e] + (count[e] + ROW_PAD - 1) / ROW_PAD * ROW_PAD;
  c->sz.n_rows = row_start[NSPEC];
  std::vector<int> row_of_atom(N), row_beg(N + 1);
  std::vector<int4> rank_info(N);
  {
    int next[NSPEC];
    for (int e = 0; e < NSPEC; ++e) next[e] = row_start[e];
    for (int i = 0; i < N; ++i) row_of_atom[i] = next[d->species[i]]++;
  }
  // systems above BRUTE_MAX atoms go through the cell list; the others are cut into K1 work items
  // (system, block of its atoms): enough items to give every SM a few CTAs, 8..64 atoms each
  std::vector<int> cell_sys, cell_cap_base(1, 0), cell_slot_base, cell_atom_list, atom_cell_sys;
  std::vector<int4> items;
  long long n_brute = 0;
  int max_brute_sys = 1;
  for (int s = 0; s < NS; ++s) {
    const int n = d->sys_offsets[s + 1] - d->sys_offsets[s];
    if (n <= BRUTE_MAX) { n_brute += n; if (n > max_brute_sys) max_brute_sys = n; }
  }
  int k1_block = (int)((n_brute / (4LL * 148) + 7) / 8 * 8);
  k1_block = k1_block < K1_MIN_BLOCK ? K1_MIN_BLOCK : k1_block > K1_MAX_BLOCK ? K1_MAX_BLOCK : k1_block;
  {
    long long beg = 0, rank_off = 0;
    for (int s = 0; s < NS; ++s) {
      const int b0 = d->sys_offsets[s], e0 = d->sys_offsets[s + 1], n = e0 - b0;
      const int cap = n - 1 < ROW_CAP ? (n - 1 > 1 ? n - 1 : 1) : ROW_CAP;
      for (int i = b0; i < e0; ++i) { row_beg[i] = (int)beg; beg += cap; }
      for (int i = b0; i < e0; ++i) {                       // rank table: (n + 31) / 32 words per atom of a brute-force system
        rank_info[i] = make_int4(n <= BRUTE_MAX ? (int)rank_off : -1, b0, n <= BRUTE_MAX ? (n + 31) / 32 : 0, 0);
        if (n <= BRUTE_MAX) rank_off += (n + 31) / 32;
      }
      if (n > BRUTE_MAX) {
        cell_slot_base.push_back((int)cell_atom_list.size());
        for (int i = b0; i < e0; ++i) { cell_atom_list.push_back(i); atom_cell_sys.push_back((int)cell_sys.size()); }
        cell_sys.push_back(s);
        cell_cap_base.push_back(cell_cap_base.back() + cells_for(n));
      } else {
        for (int a0 = b0; a0 < e0; a0 += k1_block)
          items.push_back(make_int4(b0, e0, a0, a0 + k1_block < e0 ? a0 + k1_block : e0));
        c->brute_tests += (long long)n * (n - 1);
      }
    }
    row_beg[N] = (int)beg;                              // <= cap_r: sum of n*min(128, n-1) over systems
  }
  c->n_items = (int)items.size();
  c->k1_smem = sizeof(float4) * (size_t)max_brute_sys;
  c->n_cell_sys = (int)cell_sys.size();
  c->n_cell_atoms = (int)cell_atom_list.size();
  carve(c->sz, d->workspace, &c->b);
  Buffers& b = c->b;

  // FFMA path: per element, every GEMM phase as B[k/2][n][k%2] (forward: W^T, backward: W, the last
  // one in three 128-column passes): a 16-k chunk is one contiguous bulk copy, and the two k of a
  // pair sit side by side for the packed fma.rn.f32x2 of the 32-row kernel
  std::vector<float> w((size_t)NSPEC * DEV_W_PER_ELEM, 0.0f);
  for (int e = 0; e < NSPEC; ++e) {
    const float* src = d->weights + (size_t)e * W_PER_ELEM;
    const float *W1 = src, *b1 = W1 + D1 * D0, *W2 = b1 + D1, *b2 = W2 + D2 * D1, *W3 = b2 + D2,
                *b3 = W3 + D3 * D2, *W4 = b3 + D3, *b4 = W4 + D3;
    float* dst = w.data() + (size_t)e * DEV_W_PER_ELEM;
    auto pack = [&](float* out, int K, int N, auto bval) {        // out[k/2][n][k%2] = B[k][n]: k pairs interleaved
      for (int k = 0; k < K; ++k)
        for (int n = 0; n < N; ++n) out[((size_t)(k >> 1) * N + n) * 2 + (k & 1)] = bval(k, n);
    };
    pack(dst + MLP_P_OFF0, D0, D1, [&](int k, int n) { return W1[n * D0 + k]; });
    pack(dst + MLP_P_OFF1, D1, D2, [&](int k, int n) { return W2[n * D1 + k]; });
    pack(dst + MLP_P_OFF2, D2, D3, [&](int k, int n) { return W3[n * D2 + k]; });
    pack(dst + MLP_P_OFF3, D3, D2, [&](int k, int n) { return W3[k * D2 + n]; });
    pack(dst + MLP_P_OFF4, D2, D1, [&](int k, int n) { return W2[k * D1 + n]; });
    for (int pass = 0; pass < D0 / 128; ++pass)
      pack(dst + MLP_P_OFF5 + pass * D1 * 128, D1, 128, [&](int k, int n) { return W1[k * D0 + pass * 128 + n]; });
    float* v = dst + MLP_P_FLOATS;
    memcpy(v + MLP_V_B1, b1, sizeof(float) * D1);
    memcpy(v + MLP_V_B2, b2, sizeof(float) * D2);
    memcpy(v + MLP_V_B3, b3, sizeof(float) * D3);
    memcpy(v + MLP_V_W4, W4, sizeof(float) * D3);
    v[MLP_V_B4] = b4[0];
    const float* dv = b.weights + (size_t)e * DEV_W_PER_ELEM;
    c->mlp.wpack[e] = dv;
    c->mlp.vec[e] = dv + MLP_P_FLOATS;
    c->mlp.row_end[e] = row_start[e] + count[e];
  }
  for (int e = 0; e <= NSPEC; ++e) c->mlp.row_start[e] = row_start[e];

  // cluster MLP (k3_mlp_cluster.cuh): per element and cluster rank r, the column slices [k][nc] of the six
  // phases back to back; and the table of 16-row tiles that hold real rows
  std::vector<float> wcl((size_t)NSPEC * CL_SIZE * CL_W_FLOATS);
  for (int e = 0; e < NSPEC; ++e) {
    const float* src = d->weights + (size_t)e * W_PER_ELEM;
    const float *W1 = src, *W2 = W1 + D1 * D0 + D1, *W3 = W2 + D2 * D1 + D2;
    for (int r = 0; r < CL_SIZE; ++r) {
      float* o = wcl.data() + ((size_t)e * CL_SIZE + r) * CL_W_FLOATS;
      for (int k = 0; k < D0; ++k) for (int cc = 0; cc < CL_NC0; ++cc) o[CL_W0 + k * CL_NC0 + cc] = W1[(r * CL_NC0 + cc) * D0 + k];
      for (int k = 0; k < D1; ++k) for (int cc = 0; cc < CL_NC1; ++cc) o[CL_W1 + k * CL_NC1 + cc] = W2[(r * CL_NC1 + cc) * D1 + k];
      for (int k = 0; k < D2; ++k) for (int cc = 0; cc < CL_NC2; ++cc) o[CL_W2 + k * CL_NC2 + cc] = W3[(r * CL_NC2 + cc) * D2 + k];
      for (int k = 0; k < D3; ++k) for (int cc = 0; cc < CL_NC3; ++cc) o[CL_W3 + k * CL_NC3 + cc] = W3[k * D2 + r * CL_NC3 + cc];
      for (int k = 0; k < D2; ++k) for (int cc = 0; cc < CL_NC4; ++cc) o[CL_W4 + k * CL_NC4 + cc] = W2[k * D1 + r * CL_NC4 + cc];
      for (int k = 0; k < D1; ++k) for (int cc = 0; cc < CL_NC5; ++cc) o[CL_W5 + k * CL_NC5 + cc] = W1[k * D0 + r * CL_NC5 + cc];
    }
    c->clp.vec[e] = c->mlp.vec[e];
  }
  c->clp.wcl = b.wcl;
  {
    int nt = 0;
    for (int e = 0; e < NSPEC; ++e) nt += (count[e] + CL_TM - 1) / CL_TM;
    // one wave of clusters: config 0 (22 atoms, 4 tiles) 37 -> ~10 us; beyond CL_MAX_TILES the one-CTA-per-tile
    // kernel's better per-SM efficiency wins (config 2 would need 95 clusters = 5 waves)
    c->mlp_cluster = nt <= CL_MAX_TILES && tun.k3_cluster != 1 && tun.k3_tile_rows == 0 && tun.k3_deep_ring == 0;
    if (tun.k3_cluster == 2 && nt > CL_MAX_TILES) { delete c; return PFC_ERR_ARG; }
    if (tun.k3_cluster == 2) c->mlp_cluster = true;
    c->clp.n_tiles = 0;
    if (c->mlp_cluster)
      for (int e = 0; e < NSPEC; ++e)
        for (int t = 0; t * CL_TM < count[e]; ++t) {
          const int q = c->clp.n_tiles++;
          c->clp.row0[q] = row_start[e] + t * CL_TM;
          c->clp.elem[q] = e;
          c->clp.rows[q] = count[e] - t * CL_TM < CL_TM ? count[e] - t * CL_TM : CL_TM;
        }
  }

  // tensor-core path: per element, the B operand of every phase chunk exactly as it sits in
  // shared memory -- [N rows x 32 k] fp16, K-major, SWIZZLE_64B, hi block then lo block -- with every
  // weight matrix scaled by the power of two that puts max|W| into [256, 512) (k3_mlp_tc.cuh)
  std::vector<uint8_t> wtc((size_t)NSPEC * TC_W_BYTES_PER_ELEM);
  std::vector<float> bias_tc((size_t)NSPEC * TC_BIAS_LEN, 0.0f);
  c->tc_terms = c->mlp_path == PFC_MLP_TENSOR_1TERM ? 1 : 3;
  for (int e = 0; e < NSPEC; ++e) {
    const float* src = d->weights + (size_t)e * W_PER_ELEM;
    const float *W1 = src, *b1 = W1 + D1 * D0, *W2 = b1 + D1, *b2 = W2 + D2 * D1, *W3 = b2 + D2,
                *b3 = W3 + D3 * D2, *W4 = b3 + D3, *b4 = W4 + D3;
    auto scale_log2 = [](const float* w, int n, float target) {   // e with max|w| 2^e in [target/2, target)
      float m = 0.0f;
      for (int i = 0; i < n; ++i) m = fmaxf(m, fabsf(w[i]));
      if (!(m > 0.0f) || !std::isfinite(m)) return 0;
      int ex = (int)floorf(log2f(target / m));
      return ex < -12 ? -12 : ex > 24 ? 24 : ex;
    };
    const int eW1 = scale_log2(W1, D1 * D0, 512.0f), eW2 = scale_log2(W2, D2 * D1, 512.0f),
              eW3 = scale_log2(W3, D3 * D2, 512.0f), eD = scale_log2(W4, D3, 16.0f);
    // B[n][k] of phase p (see k3_mlp_tc.cuh): forward W[n][k]; backward W[k][n]
    auto bval = [&](int p, int n, int k) -> float {
      switch (p) {
        case 0: return ldexpf(W1[n * D0 + k], eW1);
        case 1: return ldexpf(W2[n * D1 + k], eW2);
        case 2: return ldexpf(W3[n * D2 + k], eW3);
        case 3: return ldexpf(W3[k * D2 + n], eW3);
        case 4: return ldexpf(W2[k * D1 + n], eW2);
        default: return ldexpf(W1[k * D0 + (p - 5) * TC_GN + n], eW1);
      }
    };
    uint8_t* img = wtc.data() + (size_t)e * TC_W_BYTES_PER_ELEM;
    for (int p = 0; p < TC_NPHASE; ++p) {
      const int N = tc_phase_n(p), nk = tc_phase_nk(p);
      for (int ch = 0; ch < nk; ++ch) {
        uint8_t* chunk = img + tc_phase_off(p) + (size_t)ch * tc_chunk_bytes(p);
        for (int n = 0; n < N; ++n)
          for (int kk = 0; kk < TC_KC; ++kk) {
            const float v = bval(p, n, TC_KC * ch + kk);
            const __half hi = __float2half_rn(v);                       // hi: fp16 to nearest
            const __half lo = __float2half_rn(v - __half2float(hi));    // lo: the (exact) remainder, fp16 to nearest
            memcpy(chunk + tc_sw64_off(n, kk), &hi, 2);
            memcpy(chunk + (size_t)N * 64 + tc_sw64_off(n, kk), &lo, 2);
          }
      }
    }
    float* bt = bias_tc.data() + (size_t)e * TC_BIAS_LEN;
    memcpy(bt + TC_BIAS_B1, b1, sizeof(float) * D1);
    memcpy(bt + TC_BIAS_B2, b2, sizeof(float) * D2);
    memcpy(bt + TC_BIAS_B3, b3, sizeof(float) * D3);
    memcpy(bt + TC_BIAS_W4, W4, sizeof(float) * D3);
    bt[TC_BIAS_B4] = b4[0];
    for (int k = 0; k < D3; ++k) bt[TC_BIAS_W4S + k] = ldexpf(W4[k], eD);
    // epilogue factors (upload_tc_factors): inverse operand scales and the truncation compensation.  The
    // compensation scales start at the defaults and are calibrated on the handle's first batch
    // (calibrate_tc) unless pfc_tuning_t fixes them
    const int inv_scale[6] = {-(TC_AEV_SCALE_LOG2 + eW1), -eW2, -eW3, -eW3, -eW2, -(eW1 + eD)};
    for (int q = 0; q < 6; ++q) c->tc_inv_scale[e][q] = inv_scale[q];
    c->tc_lambda[e][0] = tun.tc_comp_override ? tun.tc_comp_forward : TC_LAMBDA_FWD;
    c->tc_lambda[e][1] = tun.tc_comp_override ? tun.tc_comp_backward : TC_LAMBDA_BWD;
    c->tcp.bias[e] = c->b.bias_tc + (size_t)e * TC_BIAS_LEN;
  }
  c->tcp.wpack = c->b.wtc;
  for (int e = 0; e <= NSPEC; ++e) c->tcp.row_start[e] = row_start[e];
  c->tcp.n_tiles = c->sz.n_rows / TC_TM;
  c->tcp.trace = nullptr;
  c->bias_host = bias_tc;
  // fixed by the caller, or a path that is evidence only: nothing to calibrate
  c->tc_calibrated = tun.tc_comp_override != 0 || c->mlp_path == PFC_MLP_TENSOR_1TERM;

  StepParams sp0{};
  {
    const double mass_default[NSPEC] = {1.008, 12.011, 14.007, 15.999};
    for (int e = 0; e < NSPEC; ++e) {
      const double m = d->masses_amu ? (double)d->masses_amu[e] : mass_default[e];
      if (!(m > 0.0)) { delete c; return PFC_ERR_ARG; }
      sp0.inv_mass_acc[e] = (float)(9.648533216e-3 / m);
    }
  }
  bool ok = true;
  auto up = [&](void* dst, const void* src, size_t bytes) {
    if (bytes && cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice) != cudaSuccess) ok = false;
  };
  up(b.species, d->species, sizeof(int) * N);
  up(b.sp, &sp0, sizeof(sp0));
  up(b.row_beg, row_beg.data(), sizeof(int) * (N + 1));
  up(b.rank_info, rank_info.data(), sizeof(int4) * N);
  up(b.items, items.data(), sizeof(int4) * items.size());
  up(b.sys_off, d->sys_offsets, sizeof(int) * (NS + 1));
  up(b.row_of_atom, row_of_atom.data(), sizeof(int) * N);
  up(b.weights, w.data(), sizeof(float) * w.size());
  up(b.wcl, wcl.data(), sizeof(float) * wcl.size());
  up(b.wtc, wtc.data(), wtc.size());
  up(b.bias_tc, bias_tc.data(), sizeof(float) * bias_tc.size());
  if (upload_tc_factors(c, nullptr) != PFC_OK) ok = false;
  up(b.cell_sys, cell_sys.data(), sizeof(int) * cell_sys.size());
  up(b.cell_cap_base, cell_cap_base.data(), sizeof(int) * cell_cap_base.size());
  up(b.cell_slot_base, cell_slot_base.data(), sizeof(int) * cell_slot_base.size());
  up(b.cell_atom_list, cell_atom_list.data(), sizeof(int) * cell_atom_list.size());
  up(b.atom_cell_sys, atom_cell_sys.data(), sizeof(int) * atom_cell_sys.size());
  // padded AEV rows are never written by K2: zero everything once
  if (cudaMemset(b.aev, 0, sizeof(float) * (size_t)c->sz.n_rows * AEV_LEN) != cudaSuccess) ok = false;
  if (cudaMemset(b.aev_unpacked, 0, sizeof(float) * (size_t)c->sz.n_rows * AEV_LEN) != cudaSuccess) ok = false;
  if (cudaMemset(b.status, 0, 256) != cudaSuccess) ok = false;
  if (cudaMemset(b.work, 0, 64) != cudaSuccess) ok = false;
  {
    const int skin0[4] = {1, 0, 1, 0};                  // no candidate rows yet: the first evaluation builds them; [2] = always 1
    up(b.skin_state, skin0, sizeof(skin0));
  }
  if (c->k1_smem > 48 * 1024 &&
      cudaFuncSetAttribute(k1_brute_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->k1_smem) != cudaSuccess)
    ok = false;
  if (cudaMemset(b.xlo, 0, sizeof(float4) * N) != cudaSuccess) ok = false;
#define K3_SMEM_ATTR(TM_, DEEP_)                                                                       \
  if (cudaFuncSetAttribute(k3_mlp_fp32_kernel<TM_, DEEP_>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                           (int)MlpCfg<TM_, DEEP_>::SMEM) != cudaSuccess) ok = false
  K3_SMEM_ATTR(128, false); K3_SMEM_ATTR(64, false); K3_SMEM_ATTR(32, false); K3_SMEM_ATTR(16, false);
  K3_SMEM_ATTR(32, true); K3_SMEM_ATTR(16, true);
#undef K3_SMEM_ATTR
  if (cudaFuncSetAttribute(k3_mlp_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)CL_SMEM_BYTES) != cudaSuccess) ok = false;
  if (cudaFuncSetAttribute(k3_mlp_tc_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)TC_SMEM_BYTES) != cudaSuccess) ok = false;
  if (cudaFuncSetAttribute(k3_mlp_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)TC_SMEM_BYTES) != cudaSuccess) ok = false;
  {
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && sms > 0)
      c->n_sms = sms;
  }
  {
    // FFMA K3 tile height and staging.  Measured on B200 (K3 alone): config 4, 32-row tiles, three
    // CTAs per SM, 2.11 ms; 64 rows, two CTAs per SM, 2.22 ms; 128 rows, one CTA, 2.17 ms -- and on
    // config 3 0.23 / 0.29 / 0.34 ms: co-resident small tiles hide the per-chunk latency best and
    // quantise the grid finest.  A batch that cannot give every SM a 32-row tile uses 16-row tiles
    // with the deep staging ring (config 0: 47 -> 43 us, config 2: 49 -> 45 us against two buffers;
    // with several CTAs per SM the ring is slower: config 4 2.52 ms, config 3 0.27 ms).
    // pfc_tuning_t.k3_tile_rows / k3_deep_ring override (tests reach every variant through them).
    auto tiles = [&](int tm) { int n = 0; for (int e = 0; e < NSPEC; ++e) n += (count[e] + tm - 1) / tm; return n; };
    // (16-row tiles only when they spread the batch over clearly more SMs than 32-row tiles would:
    // config 2, 95 vs 48 tiles, 47 vs 53 us; config 0 has 4 tiles either way and the packed 32-row
    // kernel takes 37 us against 45 us)
    c->mlp_tm = (tiles(32) >= c->n_sms || 2 * tiles(16) < 3 * tiles(32)) ? 32 : 16;
    c->mlp_deep = c->mlp_tm == 16;
    if (tun.k3_tile_rows) { c->mlp_tm = tun.k3_tile_rows; c->mlp_deep = false; }
    if (tun.k3_deep_ring) c->mlp_deep = tun.k3_deep_ring == 2;
    if (c->mlp_tm > 32) c->mlp_deep = false;            // the ring exists for tiles of <= 32 rows
  }
  if (cudaDeviceSynchronize() != cudaSuccess) ok = false;
  if (!ok) { cudaGetLastError(); delete c; return PFC_ERR_CUDA; }
  // launch counts (static: depends only on the configuration)
  c->launches_ef = 5 + (c->n_items > 0 ? 1 : 0) + (c->n_cell_sys > 0 ? (c->skin_list ? 7 : 5) : 0);
  c->launches_step = c->launches_ef;            // integrator kernel + forces, no energy sum inside a pfc_step call
  *out = c;
  return PFC_OK;
}

// the cached graph of this buffer triple, captured on first sight (least recently used slot evicted)
static int ef_graph(pfc_ctx* c, const float4* pos, float* E, float4* F, bool with_xlo, cudaGraphExec_t* out) {
  EfGraph* slot = &c->ef[0];
  for (EfGraph& g : c->ef) {
    if (g.exec && g.pos == pos && g.E == E && g.F == F && g.with_xlo == with_xlo) {
      g.last_use = ++c->ef_clock;
      *out = g.exec;
      return PFC_OK;
    }
    if (!g.exec) { if (slot->exec) slot = &g; }
    else if (slot->exec && g.last_use < slot->last_use) slot = &g;
  }
  if (slot->exec) { cudaGraphExecDestroy(slot->exec); slot->exec = nullptr; }
  const int rc = capture(c, 0, 1, pos, E, F, with_xlo, &slot->exec);
  if (rc != PFC_OK) return rc;
  slot->pos = pos; slot->E = E; slot->F = F; slot->with_xlo = with_xlo;
  slot->last_use = ++c->ef_clock;
  *out = slot->exec;
  return PFC_OK;
}

int pfc_energy_forces(pfc_t* c, const float* pos, float* E, float* F, void* stream) {
  if (!c || !pos || !E || !F) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  cudaStream_t st = (cudaStream_t)stream;
  // the low position words belong to the bound MD state only
  const bool with_xlo = c->bound && (const float4*)pos == c->pos;
  int rc0 = ensure_calibrated(c, (const float4*)pos, with_xlo, st);
  if (rc0 != PFC_OK) return rc0;
  cudaGraphExec_t g = nullptr;
  const int rc = ef_graph(c, (const float4*)pos, E, (float4*)F, with_xlo, &g);
  if (rc != PFC_OK) return rc;
  if (cudaGraphLaunch(g, st) != cudaSuccess) { cudaGetLastError(); return PFC_ERR_CUDA; }
  if (!c->bound) c->stream = st;
  return PFC_OK;
}

int pfc_energy_forces_nm(pfc_t* c, const float* pos_nm, float* E_kj, float* F_kj_nm, void* stream) {
  if (!c || !pos_nm || !E_kj) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  if (c->bound && (c->pos == c->b.h_pos)) return PFC_ERR_STATE;   // the staging buffers hold a pfc_run_host state
  cudaStream_t st = (cudaStream_t)stream;
  const int N = c->sz.n_atoms, NS = c->sz.n_systems;
  Buffers& b = c->b;
  k0_pack_nm_kernel<<<cdiv(N, K0_THREADS), K0_THREADS, 0, st>>>(N, pos_nm, b.h_pos);
  int rc0 = ensure_calibrated(c, b.h_pos, false, st);
  if (rc0 != PFC_OK) return rc0;
  cudaGraphExec_t g = nullptr;
  const int rc = ef_graph(c, b.h_pos, b.h_E, b.h_frc, false, &g);
  if (rc != PFC_OK) return rc;
  if (cudaGraphLaunch(g, st) != cudaSuccess) { cudaGetLastError(); return PFC_ERR_CUDA; }
  k0_unpack_kj_kernel<<<cdiv(N > NS ? N : NS, K0_THREADS), K0_THREADS, 0, st>>>(N, NS, b.h_frc, b.h_E, F_kj_nm, E_kj);
  if (!c->bound) c->stream = st;
  return cudaGetLastError() == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_profile_stages(pfc_t* c, const float* pos, float* E, float* F, void* stream, float* ms) {
  if (!c || !pos || !E || !F || !ms) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t ev[PFC_N_STAGES + 1];
  for (int k = 0; k <= PFC_N_STAGES; ++k)
    if (cudaEventCreate(&ev[k]) != cudaSuccess) return PFC_ERR_CUDA;
  {
    const int rc0 = ensure_calibrated(c, (const float4*)pos, c->bound && (const float4*)pos == c->pos, st);
    if (rc0 != PFC_OK) return rc0;
  }
  enqueue_forces(c, (const float4*)pos, E, (float4*)F, c->bound && (const float4*)pos == c->pos, st, ev);
  // stage 6: the fused integrator kernel of a steady-state step (kick + kick + drift), timed on the library's
  // staging buffers so that no caller state moves (their contents do not matter for the time; `self` is free
  // between two force evaluations and stands in for the low position words)
  if (!c->bound || c->pos != c->b.h_pos)
    LAUNCH(c, k5_verlet_kernel<2>, cdiv(c->sz.n_atoms, K5_THREADS), K5_THREADS, 0, st, c->sz.n_atoms, c->b.sp,
           c->b.species, (const float4*)F, c->b.h_pos, c->b.h_vel, c->b.self);
  cudaEventRecord(ev[PFC_N_STAGES], st);
  int rc = cudaStreamSynchronize(st) == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
  for (int k = 0; k < PFC_N_STAGES && rc == PFC_OK; ++k)
    if (cudaEventElapsedTime(&ms[k], ev[k], ev[k + 1]) != cudaSuccess) rc = PFC_ERR_CUDA;
  for (int k = 0; k <= PFC_N_STAGES; ++k) cudaEventDestroy(ev[k]);
  return rc;
}

// sums the row counts of the last evaluation: {radial entries, angular entries, triples}
__global__ void k_work_counts_kernel(int n_atoms, const int2* __restrict__ cnt, unsigned long long* __restrict__ out) {
  unsigned long long r = 0, a = 0, t = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_atoms; i += gridDim.x * blockDim.x) {
    const int2 c = cnt[i];
    r += (unsigned long long)c.x; a += (unsigned long long)c.y;
    t += (unsigned long long)((long long)c.y * (c.y - 1) / 2);
  }
  for (int o = 16; o > 0; o >>= 1) {
    r += __shfl_xor_sync(0xffffffffu, r, o); a += __shfl_xor_sync(0xffffffffu, a, o); t += __shfl_xor_sync(0xffffffffu, t, o);
  }
  if ((threadIdx.x & 31) == 0) { atomicAdd(out, r); atomicAdd(out + 1, a); atomicAdd(out + 2, t); }
}

int pfc_k3_timeline(pfc_t* c, int64_t* cycles, int32_t n) {
  if (!c || !cycles || n < 1) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  if (c->mlp_path == PFC_MLP_FP32) return PFC_ERR_STATE;
  const int total = TC_TRACE_STRIDE * TC_TRACE_ITERS;
  cudaStream_t st = c->stream;
  if (cudaMemsetAsync(c->b.trace, 0, sizeof(long long) * total, st) != cudaSuccess) return PFC_ERR_CUDA;
  TcParams tp = c->tcp;
  tp.trace = c->b.trace;
  const int grid = tp.n_tiles < c->n_sms ? tp.n_tiles : c->n_sms;
  if (c->mlp_path == PFC_MLP_TENSOR) k3_mlp_tc_kernel<3><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(tp, (const uint8_t*)c->b.aev, c->b.g, c->b.e_row);
  else k3_mlp_tc_kernel<1><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(tp, (const uint8_t*)c->b.aev, c->b.g, c->b.e_row);
  std::vector<long long> h(total);
  if (cudaMemcpyAsync(h.data(), c->b.trace, sizeof(long long) * total, cudaMemcpyDeviceToHost, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return PFC_ERR_CUDA;
  for (int i = 0; i < n && i < total; ++i) cycles[i] = (int64_t)h[i];
  return PFC_OK;
}

int pfc_work_counts(pfc_t* c, int64_t* counts) {
  if (!c || !counts) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  cudaStream_t st = c->stream;
  if (cudaMemsetAsync(c->b.work, 0, 64, st) != cudaSuccess) return PFC_ERR_CUDA;
  k_work_counts_kernel<<<148, 256, 0, st>>>(c->sz.n_atoms, c->b.cnt, c->b.work);
  unsigned long long h[3];
  if (cudaMemcpyAsync(h, c->b.work, sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return PFC_ERR_CUDA;
  counts[0] = (int64_t)h[0]; counts[1] = (int64_t)h[1]; counts[2] = (int64_t)h[2];
  counts[3] = (int64_t)c->brute_tests;
  int builds = 0;
  if (c->n_cell_sys > 0 && cudaMemcpy(&builds, c->b.skin_state + SKIN_BUILDS, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess)
    return PFC_ERR_CUDA;
  counts[4] = (int64_t)builds;
  return PFC_OK;
}

int pfc_set_state(pfc_t* c, float* pos, float* vel, float* E, float* F, void* stream) {
  if (!c || !pos || !vel || !E || !F) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  cudaStream_t st = (cudaStream_t)stream;
  const bool same = c->bound && c->pos == (float4*)pos && c->vel == (float4*)vel && c->E == E &&
                    c->frc == (float4*)F;
  if (!same) drop_state_graphs(c);                 // pointers are baked into the graphs
  c->pos = (float4*)pos; c->vel = (float4*)vel; c->E = E; c->frc = (float4*)F;
  c->stream = st;
  c->bound = true;
  c->forces_stale = true;
  c->steps_total = 0;
  k5_reset_counter_kernel<<<1, 1, 0, st>>>(c->b.sp);
  if (cudaMemsetAsync(c->b.xlo, 0, sizeof(float4) * c->sz.n_atoms, st) != cudaSuccess) return PFC_ERR_CUDA;
  return PFC_OK;
}

// after step `steps_total` (1-based) of the bound state: positions x_n are final once the step's
// drift kernel and force graph are enqueued -- store a frame every frame_stride steps
static int maybe_store_frame(pfc_ctx* c, cudaStream_t st) {
  ++c->steps_total;
  if (!c->frames || c->frame_stride <= 0 || c->steps_total % c->frame_stride != 0) return PFC_OK;
  if (c->frames_written >= c->frame_cap) return PFC_OK;
  const size_t nb = sizeof(float4) * (size_t)c->sz.n_atoms;
  if (cudaMemcpyAsync(c->frames + (size_t)c->frames_written * c->sz.n_atoms, c->pos, nb, cudaMemcpyDeviceToDevice,
                      st) != cudaSuccess)
    return PFC_ERR_CUDA;
  ++c->frames_written;
  return PFC_OK;
}

// steps until (and including) the next one after which a frame is due; a huge number if none
static long long steps_to_next_frame(const pfc_ctx* c) {
  if (!c->frames || c->frame_stride <= 0 || c->frames_written >= c->frame_cap) return 1LL << 60;
  return c->frame_stride - (c->steps_total % c->frame_stride);
}

static int run_steps(pfc_ctx* c, int32_t n_steps, float dt_fs, bool langevin) {
  cudaStream_t st = c->stream;
  int rc;
  const int kind = langevin ? 2 : 1;
  if ((rc = ensure_calibrated(c, c->pos, true, st)) != PFC_OK) return rc;   // before anything is captured
  if (!c->g_forces && (rc = capture(c, 0, 1, c->pos, c->E, c->frc, true, &c->g_forces)) != PFC_OK) return rc;
  cudaGraphExec_t* g1 = langevin ? &c->g_lstep : &c->g_step;
  cudaGraphExec_t* gk = langevin ? &c->g_lstepk : &c->g_stepk;
  if (!*g1 && (rc = capture(c, kind, 1, c->pos, c->E, c->frc, true, g1)) != PFC_OK) return rc;
  const int K = c->steps_per_graph;
  if (K > 1 && n_steps - 1 >= K && !*gk && (rc = capture(c, kind, K, c->pos, c->E, c->frc, true, gk)) != PFC_OK)
    return rc;
  if (dt_fs != c->cur_dt) {
    k5_set_params_kernel<<<1, 1, 0, st>>>(c->b.sp, dt_fs);
    c->cur_dt = dt_fs;
  }
  if (c->forces_stale) {
    if (cudaGraphLaunch(c->g_forces, st) != cudaSuccess) return PFC_ERR_CUDA;
    c->forces_stale = false;
  }
  if (n_steps == 0) return PFC_OK;
  // step 1: half kick + drift, forces.  steps 2..n: fused (trailing half kick + leading half kick +
  // drift), forces -- K of them per graph launch while no frame falls inside the span, else one per
  // launch.  Then the last half kick and the per-system energies of the final state (the step graphs
  // leave the energy sum out: E cannot be read between the steps of one call).
  if (langevin) enqueue_langevin<1>(c, st); else enqueue_verlet<1>(c, st);
  if (n_steps == 1 && c->early_pos_dst) {            // x_1 is final: its copy to the host overlaps the force evaluation
    if (cudaEventRecord(c->ev_drift, st) != cudaSuccess || cudaStreamWaitEvent(c->copy_stream, c->ev_drift, 0) != cudaSuccess ||
        cudaMemcpyAsync(c->early_pos_dst, c->pos, sizeof(float4) * (size_t)c->sz.n_atoms, cudaMemcpyDeviceToHost,
                        c->copy_stream) != cudaSuccess ||
        cudaEventRecord(c->ev_copied, c->copy_stream) != cudaSuccess)
      return PFC_ERR_CUDA;
  }
  if (cudaGraphLaunch(c->g_forces, st) != cudaSuccess) return PFC_ERR_CUDA;
  if ((rc = maybe_store_frame(c, st)) != PFC_OK) return rc;
  int left = n_steps - 1;
  while (left > 0) {
    if (*gk && left >= K && steps_to_next_frame(c) >= K) {
      if (cudaGraphLaunch(*gk, st) != cudaSuccess) return PFC_ERR_CUDA;
      c->steps_total += K - 1;                       // (no frame is due inside the span)
      if ((rc = maybe_store_frame(c, st)) != PFC_OK) return rc;
      left -= K;
    } else {
      if (cudaGraphLaunch(*g1, st) != cudaSuccess) return PFC_ERR_CUDA;
      if ((rc = maybe_store_frame(c, st)) != PFC_OK) return rc;
      --left;
    }
  }
  enqueue_verlet<0>(c, st);
  if (n_steps > 1) enqueue_energy_sum(c, c->frc, c->E, st);   // (n_steps == 1: the force graph of step 1 has summed)
  return cudaGetLastError() == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_step(pfc_t* c, int32_t n_steps, float dt_fs) {
  if (!c || n_steps < 0 || !(dt_fs > 0.0f)) return PFC_ERR_ARG;
  if (!c->bound || !on_device(c)) return PFC_ERR_STATE;
  return run_steps(c, n_steps, dt_fs, false);
}

int pfc_step_langevin(pfc_t* c, int32_t n_steps, float dt_fs, float friction_per_fs, float temperature_K,
                      uint64_t seed) {
  if (!c || n_steps < 0 || !(dt_fs > 0.0f) || !(friction_per_fs >= 0.0f) || !(temperature_K >= 0.0f))
    return PFC_ERR_ARG;
  if (!c->bound || !on_device(c)) return PFC_ERR_STATE;
  if (friction_per_fs != c->lg_gamma || temperature_K != c->lg_T || dt_fs != c->lg_dt || seed != c->lg_seed) {
    const double c1 = exp(-(double)friction_per_fs * (double)dt_fs), c2 = sqrt(1.0 - c1 * c1);
    k5_set_langevin_kernel<<<1, 1, 0, c->stream>>>(c->b.sp, (float)c1, (float)c2,
                                                    (float)(8.617333262e-5 * (double)temperature_K),
                                                    (uint32_t)seed, (uint32_t)(seed >> 32));
    c->lg_gamma = friction_per_fs; c->lg_T = temperature_K; c->lg_dt = dt_fs; c->lg_seed = seed;
  }
  return run_steps(c, n_steps, dt_fs, true);
}

int pfc_set_frames(pfc_t* c, float* frames, int32_t stride, int32_t max_frames) {
  if (!c || stride < 0 || max_frames < 0 || (frames && (stride < 1 || max_frames < 1))) return PFC_ERR_ARG;
  c->frames = (float4*)frames;
  c->frame_stride = frames ? stride : 0;
  c->frame_cap = frames ? max_frames : 0;
  c->frames_written = 0;
  return PFC_OK;
}

int pfc_frames_written(pfc_t* c, int32_t* n) {
  if (!c || !n) return PFC_ERR_ARG;
  *n = c->frames_written;
  return PFC_OK;
}

static int run_host_impl(pfc_t* c, float* pos_h, float* vel_h, int32_t n_steps, float dt_fs, float* E_h,
                         float* F_h, void* stream, bool forces_in) {
  if (!c || !pos_h || !vel_h || !E_h || (forces_in && !F_h)) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nb = sizeof(float4) * (size_t)c->sz.n_atoms;
  Buffers& b = c->b;
  if (cudaMemcpyAsync(b.h_pos, pos_h, nb, cudaMemcpyHostToDevice, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaMemcpyAsync(b.h_vel, vel_h, nb, cudaMemcpyHostToDevice, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (forces_in && cudaMemcpyAsync(b.h_frc, F_h, nb, cudaMemcpyHostToDevice, st) != cudaSuccess) return PFC_ERR_CUDA;
  int rc = pfc_set_state(c, (float*)b.h_pos, (float*)b.h_vel, b.h_E, (float*)b.h_frc, stream);
  if (rc != PFC_OK) return rc;
  if (forces_in) c->forces_stale = false;          // the caller vouches: F_h = forces at pos_h
  // one step with known forces: the new positions are final after the first kernel -- copy them back meanwhile
  const bool early = forces_in && n_steps == 1;
  if (early && !c->copy_stream) {
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_drift, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_copied, cudaEventDisableTiming) != cudaSuccess)
      return PFC_ERR_CUDA;
  }
  c->early_pos_dst = early ? (float4*)pos_h : nullptr;
  rc = pfc_step(c, n_steps, dt_fs);
  c->early_pos_dst = nullptr;
  if (rc != PFC_OK) return rc;
  if (early) {
    if (cudaStreamWaitEvent(st, c->ev_copied, 0) != cudaSuccess) return PFC_ERR_CUDA;
  } else if (cudaMemcpyAsync(pos_h, b.h_pos, nb, cudaMemcpyDeviceToHost, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaMemcpyAsync(vel_h, b.h_vel, nb, cudaMemcpyDeviceToHost, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (F_h && cudaMemcpyAsync(F_h, b.h_frc, nb, cudaMemcpyDeviceToHost, st) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaMemcpyAsync(E_h, b.h_E, sizeof(float) * c->sz.n_systems, cudaMemcpyDeviceToHost, st) != cudaSuccess)
    return PFC_ERR_CUDA;
  return cudaStreamSynchronize(st) == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_run_host(pfc_t* c, float* pos_h, float* vel_h, int32_t n_steps, float dt_fs, float* E_h, float* F_h,
                 void* stream) {
  return run_host_impl(c, pos_h, vel_h, n_steps, dt_fs, E_h, F_h, stream, false);
}

int pfc_run_host_resume(pfc_t* c, float* pos_h, float* vel_h, float* F_h, int32_t n_steps, float dt_fs,
                        float* E_h, void* stream) {
  return run_host_impl(c, pos_h, vel_h, n_steps, dt_fs, E_h, F_h, stream, true);
}

int pfc_get_neighbors(pfc_t* c, const int32_t** r_off, const int32_t** r_idx, const int32_t** a_off,
                      const int32_t** a_idx) {
  if (!c) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  // export the step path's fixed-capacity rows into the canonical CSR (reading S7)
  const Sizes& s = c->sz;
  const Buffers& b = c->b;
  cudaStream_t st = c->stream;
  if (s.n_scan_blocks > 1) k1_scan_totals_kernel<<<s.n_scan_blocks, SCAN_THREADS, 0, st>>>(s.n_atoms, b.cnt, b.block_tot);
  k1_scan_kernel<<<s.n_scan_blocks, SCAN_THREADS, 0, st>>>(s.n_atoms, b.cnt, b.block_tot, b.r_off, b.a_off);
  k1_export_csr_kernel<<<cdiv(s.n_atoms, K1_WARPS), K1_WARPS * 32, 0, st>>>(s.n_atoms, b.row_beg, b.nbr, b.cnt, b.r_off,
                                                                          b.a_off, b.r_idx, b.a_idx);
  // the export overwrote the block that holds the candidate rows of cell-list systems: rebuild them next time
  if (c->n_cell_sys > 0 && c->skin_list) k1_skin_invalidate_kernel<<<1, 1, 0, st>>>(b.skin_state);
  if (cudaGetLastError() != cudaSuccess) return PFC_ERR_CUDA;
  if (r_off) *r_off = b.r_off;
  if (r_idx) *r_idx = b.r_idx;
  if (a_off) *a_off = b.a_off;
  if (a_idx) *a_idx = b.a_idx;
  return PFC_OK;
}

// ---- the entry point with static scratch (include/pfc_noalloc.h) ----------------------------------
// Block totals of the reduce-then-scan over cnt: one int2 per SCAN_BLOCK atoms.  A file-scope device
// array: resident on every GPU that loads the library; shared by all calls (they race if they overlap).
constexpr int NOALLOC_MAX_BLOCKS = PFC_NOALLOC_MAX_ATOMS / SCAN_BLOCK;
static_assert(NOALLOC_MAX_BLOCKS * SCAN_BLOCK == PFC_NOALLOC_MAX_ATOMS && NOALLOC_MAX_BLOCKS == 512, "static scratch size");
static __device__ __align__(256) int2 g_noalloc_block_tot[NOALLOC_MAX_BLOCKS];

// In host code the array's name is a stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
constexpr int NOALLOC_MAX_DEVICES = 64;
static int2* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};
static std::mutex g_noalloc_mutex;

static int noalloc_scratch(int device, int2** out) {
  if (device < 0 || device >= NOALLOC_MAX_DEVICES) return PFC_ERR_STATE;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[device]) {
    int2* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_noalloc_block_tot) != cudaSuccess || !p) { cudaGetLastError(); return PFC_ERR_CUDA; }
    g_noalloc_ptr[device] = p;
  }
  *out = g_noalloc_ptr[device];
  return PFC_OK;
}

int pfc_neighbor_offsets_noalloc(pfc_t* c, int32_t* r_off, int32_t* a_off, void* stream) {
  if (!c || !r_off || !a_off) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;            // (so the symbol address below belongs to the handle's device)
  if (c->sz.n_atoms > PFC_NOALLOC_MAX_ATOMS) return PFC_ERR_TOO_LARGE;
  int2* tot = nullptr;
  const int rc = noalloc_scratch(c->device, &tot);
  if (rc != PFC_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int n = c->sz.n_atoms, nb = cdiv(n, SCAN_BLOCK);
  // the same two kernels as the export of pfc_get_neighbors, their block totals in the static array
  // (block q's total is written by the first kernel before the second reads totals 0 .. q-1)
  if (nb > 1) k1_scan_totals_kernel<<<nb, SCAN_THREADS, 0, st>>>(n, c->b.cnt, tot);
  k1_scan_kernel<<<nb, SCAN_THREADS, 0, st>>>(n, c->b.cnt, tot, r_off, a_off);
  return cudaGetLastError() == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_get_intermediates(pfc_t* c, const float** aev, const float** g, const int32_t** row_of_atom,
                          int32_t* n_rows) {
  if (!c) return PFC_ERR_ARG;
  if (aev) {
    if (c->mlp_path == PFC_MLP_FP32) {
      *aev = c->b.aev;
    } else {                                            // the tensor path keeps the AEV as the packed operand image: unpack it
      if (!on_device(c)) return PFC_ERR_STATE;
      const int n = c->sz.n_rows * AEV_LEN;
      k2_unpack16_kernel<<<cdiv(n, 256), 256, 0, c->stream>>>(c->sz.n_rows, (const uint8_t*)c->b.aev, c->b.aev_unpacked);
      if (cudaGetLastError() != cudaSuccess) return PFC_ERR_CUDA;
      *aev = c->b.aev_unpacked;
    }
  }
  if (g) *g = c->b.g;
  if (row_of_atom) *row_of_atom = c->b.row_of_atom;
  if (n_rows) *n_rows = c->sz.n_rows;
  return PFC_OK;
}

int pfc_copy_to_host(const void* src, void* dst, size_t bytes) {
  if (!src || !dst) return PFC_ERR_ARG;
  return cudaMemcpy(dst, src, bytes, cudaMemcpyDeviceToHost) == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_status(pfc_t* c, uint32_t* bits) {
  if (!c || !bits) return PFC_ERR_ARG;
  if (!on_device(c)) return PFC_ERR_STATE;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return PFC_ERR_CUDA;
  if (cudaMemcpy(bits, c->b.status, sizeof(uint32_t), cudaMemcpyDeviceToHost) != cudaSuccess) return PFC_ERR_CUDA;
  return PFC_OK;
}

int pfc_tc_chain_probe(const float* A, const float* B, int32_t n_slices, int32_t n_mma, float* D, void* stream) {
  if (!A || !B || !D || n_slices < 1 || n_slices > TCP_MAX_SLICES || n_mma < 1 || n_mma > 4096) return PFC_ERR_ARG;
  const size_t smem = 1024 + (size_t)((n_slices + 1) / 2) * (TCP_M + TCP_N) * 64;
  if (cudaFuncSetAttribute(tc_chain_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
    cudaGetLastError();
    return PFC_ERR_CUDA;
  }
  tc_chain_probe_kernel<<<1, 128, smem, (cudaStream_t)stream>>>(A, B, n_slices, n_mma, D);
  return cudaGetLastError() == cudaSuccess ? PFC_OK : PFC_ERR_CUDA;
}

int pfc_tc_calibration(pfc_t* c, float* out) {
  if (!c || !out) return PFC_ERR_ARG;
  for (int e = 0; e < NSPEC; ++e) {
    out[8 * e + 0] = c->tc_lambda[e][0]; out[8 * e + 1] = c->tc_lambda[e][1];
    for (int k = 0; k < 4; ++k) out[8 * e + 2 + k] = c->tc_resid[e][k];
    out[8 * e + 6] = c->tc_calibrated ? 1.0f : 0.0f;
    out[8 * e + 7] = (float)c->tc_fallback;
  }
  return PFC_OK;
}

int pfc_mlp_path(pfc_t* c, int32_t* path) {
  if (!c || !path) return PFC_ERR_ARG;
  *path = c->mlp_path;
  return PFC_OK;
}

int pfc_launch_counts(pfc_t* c, int32_t* per_ef, int32_t* per_step, int32_t* steps_per_graph) {
  if (!c) return PFC_ERR_ARG;
  if (per_ef) *per_ef = c->launches_ef;
  if (per_step) *per_step = c->launches_step;
  if (steps_per_graph) *steps_per_graph = c->steps_per_graph;
  return PFC_OK;
}

int pfc_destroy(pfc_t* c) {
  if (!c) return PFC_ERR_ARG;
  drop_state_graphs(c);
  for (EfGraph& g : c->ef)
    if (g.exec) cudaGraphExecDestroy(g.exec);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->ev_drift) cudaEventDestroy(c->ev_drift);
  if (c->ev_copied) cudaEventDestroy(c->ev_copied);
  delete c;
  return PFC_OK;
}

const char* pfc_error_string(int code) {
  switch (code) {
    case PFC_OK: return "ok";
    case PFC_ERR_ARG: return "invalid argument";
    case PFC_ERR_SPECIES: return "species outside 0..3 or malformed sys_offsets";
    case PFC_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case PFC_ERR_CUDA: return "CUDA runtime error";
    case PFC_ERR_CAPTURE: return "CUDA graph capture failed";
    case PFC_ERR_STATE: return "no MD state bound (pfc_set_state), or the handle's CUDA device is not current";
    case PFC_ERR_TOO_LARGE: return "the handle has more atoms than the static scratch of the no-allocation entry point holds (PFC_NOALLOC_MAX_ATOMS)";
    default: return "unknown pfc error";
  }
}

}  // extern "C"
