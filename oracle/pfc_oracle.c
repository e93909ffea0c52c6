/* pfc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU definition of what the `pfc` hot path computes:
 * neighbour lists, ANI-style atomic environment vectors (AEV), per-element
 * MLP energy, forces F = -dE/dx by the explicitly written chain rule, and the
 * velocity-Verlet map.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with paper_2412_18271_b200/csrc (the CUDA path).
 *
 * What it follows.  The paper fixes only the contract: positions in,
 * scalar energy out, forces by differentiation, NVE
 * integration from 300 K velocities.  It prints no formula for a
 * potential.  The potential is the one BASELINE.json:configs[0] names,
 * completed as SURVEY.md section 8(c) O1-O8 with the readings S1-S24 (restated
 * in DESIGN.md).  Each function below cites the O-step it writes out.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1/P2 golden values
 * (tests/golden/), P3 finite differences, P4 invariances, P5 torch fp64
 * celu/matmul/autograd, P6 independent torch-autograd AEV, P7 brute-force vs
 * cell list, P8 dt^2 NVE error, P9 reversibility, P10 harmonic oscillator;
 * O9 (Langevin, at the end of this file): P13 Philox known-answer vectors, P14
 * moments of the normals, P15 zero friction = O8, P16 free-particle
 * thermalisation (tests/test_oracle_langevin.py).
 * P12: absolute energies of this random-weight potential are "parity
 * unpinned" beyond those (no printed value exists anywhere).
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC (see
 * oracle/__init__.py).  -ffp-contract=off matters: the cutoff predicate (O2)
 * is DEFINED as individually rounded fp32 operations.
 */
#include <float.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#if defined(FLT_EVAL_METHOD) && FLT_EVAL_METHOD != 0
#error "float expressions must be evaluated in float (O2 predicate)"
#endif

/* ---- model constants: fp32 literals promoted to double (S8) --------------- */
#define NSPEC 4
#define NSHF_R 16
#define NSHF_A 4
#define NSHF_Z 8
#define NPAIR 10
#define RAD_LEN (NSPEC * NSHF_R)                 /* 64  */
#define ANG_LEN (NPAIR * NSHF_A * NSHF_Z)        /* 320 */
#define AEV_LEN (RAD_LEN + ANG_LEN)              /* 384 */
#define D1 160
#define D2 128
#define D3 96
#define W_PER_ELEM (D1 * AEV_LEN + D1 + D2 * D1 + D2 + D3 * D2 + D3 + D3 + 1) /* 94689 */

static const float RC2_R_F = 27.04f;             /* S6: 0x41d851ec, not 5.2f*5.2f */
static const float RC2_A_F = 12.25f;
static const double RC_R = (double)5.2f;
static const double RC_A = (double)3.5f;
static const double ETA_R = (double)16.0f;
static const double ETA_A = (double)8.0f;
static const double COS_SCALE = (double)0.95f;   /* S5 */
static const double ALPHA = (double)0.1f;        /* CELU */
static const double PI = 3.14159265358979323846;
static const double ACC = 9.648533216e-3;        /* (A/fs^2) per (eV/A/amu) */
static const float SHF_R_F[NSHF_R] = {           /* S2: 0.9 + k*0.26875 */
    0.9f, 1.16875f, 1.4375f, 1.70625f, 1.975f, 2.24375f, 2.5125f, 2.78125f,
    3.05f, 3.31875f, 3.5875f, 3.85625f, 4.125f, 4.39375f, 4.6625f, 4.93125f};
static const float SHF_A_F[NSHF_A] = {0.9f, 1.55f, 2.2f, 2.85f};   /* S3 */
static const float SHF_Z_F[NSHF_Z] = {           /* S3: pi/16 + b*pi/8 */
    0.19634954f, 0.58904862f, 0.98174770f, 1.37444679f,
    1.76714587f, 2.15984495f, 2.55254403f, 2.94524311f};

int oracle_aev_len(void) { return AEV_LEN; }
int oracle_weights_per_element(void) { return W_PER_ELEM; }
int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- O2: the cutoff predicate, fp32, individually rounded, no FMA ---------- */
static float dist2_f32(const float *a, const float *b) {
    float dx = a[0] - b[0];
    float dy = a[1] - b[1];
    float dz = a[2] - b[2];
    float xx = dx * dx;
    float yy = dy * dy;
    float zz = dz * dz;
    float s = xx + yy;
    s = s + zz;
    return s;
}
/* exported so a test can check that the build did not contract a*b+c */
float oracle_dist2_f32(const float *a, const float *b) { return dist2_f32(a, b); }

static int system_of(const int32_t *sys_off, int n_sys, int i) {
    int lo = 0, hi = n_sys;               /* largest s with sys_off[s] <= i */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (sys_off[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

/* O2, O(N^2) enumeration.  pos is fp32 [N][3].  Rows ascending in j; j ranges
 * over the atoms of i's own system only (S22).  If r_idx == NULL only the
 * offsets (row counts) are produced.  Returns 0, or -1 if a capacity is short. */
int oracle_neighbors(int n_atoms, int n_sys, const int32_t *sys_off, const float *pos,
                     int32_t *r_off, int32_t *r_idx, int64_t cap_r,
                     int32_t *a_off, int32_t *a_idx, int64_t cap_a) {
    int fill = (r_idx != NULL);
    if (!fill) {
        r_off[0] = 0; a_off[0] = 0;
#pragma omp parallel for schedule(dynamic, 64)
        for (int i = 0; i < n_atoms; ++i) {
            int s = system_of(sys_off, n_sys, i);
            int nr = 0, na = 0;
            for (int j = sys_off[s]; j < sys_off[s + 1]; ++j) {
                if (j == i) continue;
                float d2 = dist2_f32(pos + 3 * i, pos + 3 * j);
                if (d2 < RC2_R_F) ++nr;
                if (d2 < RC2_A_F) ++na;
            }
            r_off[i + 1] = nr; a_off[i + 1] = na;
        }
        for (int i = 0; i < n_atoms; ++i) {       /* counts -> offsets */
            r_off[i + 1] += r_off[i];
            a_off[i + 1] += a_off[i];
        }
        return 0;
    }
    if (r_off[n_atoms] > cap_r || a_off[n_atoms] > cap_a) return -1;
#pragma omp parallel for schedule(dynamic, 64)
    for (int i = 0; i < n_atoms; ++i) {
        int s = system_of(sys_off, n_sys, i);
        int32_t *rr = r_idx + r_off[i], *aa = a_idx + a_off[i];
        for (int j = sys_off[s]; j < sys_off[s + 1]; ++j) {
            if (j == i) continue;
            float d2 = dist2_f32(pos + 3 * i, pos + 3 * j);
            if (d2 < RC2_R_F) *rr++ = j;
            if (d2 < RC2_A_F) *aa++ = j;
        }
    }
    return 0;
}

static int cmp_i32(const void *a, const void *b) {
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* O2 through a cell list (pin P7 demands it reproduce oracle_neighbors
 * exactly).  Cells of edge >= cell_edge (> 5.2) over each system's bounding
 * box; the SAME fp32 predicate decides membership; rows sorted ascending. */
int oracle_neighbors_cell(int n_atoms, int n_sys, const int32_t *sys_off, const float *pos,
                          double cell_edge,
                          int32_t *r_off, int32_t *r_idx, int64_t cap_r,
                          int32_t *a_off, int32_t *a_idx, int64_t cap_a) {
    int fill = (r_idx != NULL);
    if (!fill) { r_off[0] = 0; a_off[0] = 0; }
    else if (r_off[n_atoms] > cap_r || a_off[n_atoms] > cap_a) return -1;
    for (int s = 0; s < n_sys; ++s) {
        int b = sys_off[s], e = sys_off[s + 1], n = e - b;
        if (n <= 0) continue;
        double lo[3], hi[3];
        for (int d = 0; d < 3; ++d) { lo[d] = hi[d] = pos[3 * b + d]; }
        for (int i = b; i < e; ++i)
            for (int d = 0; d < 3; ++d) {
                double v = pos[3 * i + d];
                if (v < lo[d]) lo[d] = v;
                if (v > hi[d]) hi[d] = v;
            }
        int nc[3];
        for (int d = 0; d < 3; ++d) {
            nc[d] = (int)floor((hi[d] - lo[d]) / cell_edge) + 1;
            if (nc[d] > 256) nc[d] = 256;
        }
        double ce[3];
        for (int d = 0; d < 3; ++d) {
            ce[d] = (hi[d] - lo[d]) / nc[d];
            if (ce[d] < cell_edge) ce[d] = cell_edge;
        }
        int ncell = nc[0] * nc[1] * nc[2];
        int32_t *head = (int32_t *)malloc(sizeof(int32_t) * (size_t)(ncell + 1));
        int32_t *cell_of = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
        int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
        memset(head, 0, sizeof(int32_t) * (size_t)(ncell + 1));
        for (int i = b; i < e; ++i) {
            int c[3];
            for (int d = 0; d < 3; ++d) {
                c[d] = (int)floor((pos[3 * i + d] - lo[d]) / ce[d]);
                if (c[d] < 0) c[d] = 0;
                if (c[d] >= nc[d]) c[d] = nc[d] - 1;
            }
            cell_of[i - b] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
            head[cell_of[i - b] + 1]++;
        }
        for (int c = 0; c < ncell; ++c) head[c + 1] += head[c];
        int32_t *cursor = (int32_t *)malloc(sizeof(int32_t) * (size_t)ncell);
        memcpy(cursor, head, sizeof(int32_t) * (size_t)ncell);
        for (int i = b; i < e; ++i) order[cursor[cell_of[i - b]]++] = i;
        free(cursor);
#pragma omp parallel
        {
            int32_t *tmp_r = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
            int32_t *tmp_a = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
#pragma omp for schedule(dynamic, 64)
            for (int i = b; i < e; ++i) {
                int ci = cell_of[i - b];
                int cx = ci % nc[0], cy = (ci / nc[0]) % nc[1], cz = ci / (nc[0] * nc[1]);
                int nr = 0, na = 0;
                for (int z = cz - 1; z <= cz + 1; ++z) {
                    if (z < 0 || z >= nc[2]) continue;
                    for (int y = cy - 1; y <= cy + 1; ++y) {
                        if (y < 0 || y >= nc[1]) continue;
                        for (int x = cx - 1; x <= cx + 1; ++x) {
                            if (x < 0 || x >= nc[0]) continue;
                            int c = (z * nc[1] + y) * nc[0] + x;
                            for (int q = head[c]; q < head[c + 1]; ++q) {
                                int j = order[q];
                                if (j == i) continue;
                                float d2 = dist2_f32(pos + 3 * i, pos + 3 * j);
                                if (d2 < RC2_R_F) tmp_r[nr++] = j;
                                if (d2 < RC2_A_F) tmp_a[na++] = j;
                            }
                        }
                    }
                }
                if (!fill) { r_off[i + 1] = nr; a_off[i + 1] = na; }
                else {
                    qsort(tmp_r, (size_t)nr, sizeof(int32_t), cmp_i32);
                    qsort(tmp_a, (size_t)na, sizeof(int32_t), cmp_i32);
                    memcpy(r_idx + r_off[i], tmp_r, sizeof(int32_t) * (size_t)nr);
                    memcpy(a_idx + a_off[i], tmp_a, sizeof(int32_t) * (size_t)na);
                }
            }
            free(tmp_r); free(tmp_a);
        }
        free(head); free(cell_of); free(order);
    }
    if (!fill)
        for (int i = 0; i < n_atoms; ++i) {
            r_off[i + 1] += r_off[i];
            a_off[i + 1] += a_off[i];
        }
    return 0;
}

/* ---- O3/O4: symmetry functions -------------------------------------------- */
static double fcut(double r, double rc) { return 0.5 * cos(PI * r / rc) + 0.5; }
static double dfcut(double r, double rc) { return -(PI / (2.0 * rc)) * sin(PI * r / rc); }

/* species-pair block index p (O4): HH0 HC1 HN2 HO3 CC4 CN5 CO6 NN7 NO8 OO9 */
static int pair_index(int za, int zb) {
    int s1 = za < zb ? za : zb, s2 = za < zb ? zb : za;
    return s1 * NSPEC - s1 * (s1 - 1) / 2 + (s2 - s1);
}
int oracle_pair_index(int za, int zb) { return pair_index(za, zb); }

/* AEV of centre i (O3 radial, O4 angular).  rj/aj: global indices of its
 * radial / angular neighbours.  pos fp64 [N][3]. */
static void atom_aev(const double *pos, const int32_t *species, int i,
                     const int32_t *rj, int nr, const int32_t *aj, int na, double *aev) {
    for (int a = 0; a < AEV_LEN; ++a) aev[a] = 0.0;
    const double *xi = pos + 3 * i;
    for (int n = 0; n < nr; ++n) {                       /* O3 */
        int j = rj[n];
        double d[3] = {pos[3 * j] - xi[0], pos[3 * j + 1] - xi[1], pos[3 * j + 2] - xi[2]};
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double fc = fcut(r, RC_R);
        for (int k = 0; k < NSHF_R; ++k) {
            double dr = r - (double)SHF_R_F[k];
            aev[NSHF_R * species[j] + k] += 0.25 * exp(-ETA_R * dr * dr) * fc;
        }
    }
    for (int n = 0; n < na; ++n) {                       /* O4: unordered pairs n<m */
        int j = aj[n];
        double vj[3] = {pos[3 * j] - xi[0], pos[3 * j + 1] - xi[1], pos[3 * j + 2] - xi[2]};
        double rjn = sqrt(vj[0] * vj[0] + vj[1] * vj[1] + vj[2] * vj[2]);
        for (int m = n + 1; m < na; ++m) {
            int k = aj[m];
            double vk[3] = {pos[3 * k] - xi[0], pos[3 * k + 1] - xi[1], pos[3 * k + 2] - xi[2]};
            double rkn = sqrt(vk[0] * vk[0] + vk[1] * vk[1] + vk[2] * vk[2]);
            double cosphi = (vj[0] * vk[0] + vj[1] * vk[1] + vj[2] * vk[2]) / (rjn * rkn);
            double theta = acos(COS_SCALE * cosphi);
            double rbar = 0.5 * (rjn + rkn);
            double fcc = fcut(rjn, RC_A) * fcut(rkn, RC_A);
            int p = pair_index(species[j], species[k]);
            double A[NSHF_Z];                            /* angular factor, same for every a */
            for (int b = 0; b < NSHF_Z; ++b)
                A[b] = pow(0.5 * (1.0 + cos(theta - (double)SHF_Z_F[b])), 32.0);
            for (int a = 0; a < NSHF_A; ++a) {
                double dr = rbar - (double)SHF_A_F[a];
                double B = exp(-ETA_A * dr * dr);
                for (int b = 0; b < NSHF_Z; ++b)
                    aev[RAD_LEN + 32 * p + 8 * a + b] += 2.0 * A[b] * B * fcc;
            }
        }
    }
}

/* ---- O5: per-element MLP, forward and input gradient ----------------------- */
static double celu(double x) {
    /* CELU(x) = max(0,x) + min(0, alpha*(exp(min(x,0)/alpha) - 1)) */
    double xp = x > 0.0 ? x : 0.0;
    double xm = x < 0.0 ? x : 0.0;
    double neg = ALPHA * expm1(xm / ALPHA);
    return xp + (neg < 0.0 ? neg : 0.0);
}
static double dcelu(double x) { return x > 0.0 ? 1.0 : exp(x / ALPHA); }

/* weights of one element (fp32, promoted): W1[160][384] b1 W2[128][160] b2
 * W3[96][128] b3 W4[1][96] b4.  e = energy of the atom, g = de/daev. */
static void mlp_fwd_bwd(const float *w, const double *aev, double *e_out, double *g) {
    const float *W1 = w, *b1 = W1 + D1 * AEV_LEN, *W2 = b1 + D1, *b2 = W2 + D2 * D1,
                *W3 = b2 + D2, *b3 = W3 + D3 * D2, *W4 = b3 + D3, *b4 = W4 + D3;
    double z1[D1], h1[D1], z2[D2], h2[D2], z3[D3], h3[D3];
    for (int o = 0; o < D1; ++o) {
        double s = (double)b1[o];
        for (int k = 0; k < AEV_LEN; ++k) s += (double)W1[o * AEV_LEN + k] * aev[k];
        z1[o] = s; h1[o] = celu(s);
    }
    for (int o = 0; o < D2; ++o) {
        double s = (double)b2[o];
        for (int k = 0; k < D1; ++k) s += (double)W2[o * D1 + k] * h1[k];
        z2[o] = s; h2[o] = celu(s);
    }
    for (int o = 0; o < D3; ++o) {
        double s = (double)b3[o];
        for (int k = 0; k < D2; ++k) s += (double)W3[o * D2 + k] * h2[k];
        z3[o] = s; h3[o] = celu(s);
    }
    double e = (double)b4[0];
    for (int k = 0; k < D3; ++k) e += (double)W4[k] * h3[k];
    *e_out = e;
    if (!g) return;
    double d3[D3], d2[D2], d1[D1];                       /* de/dz of each layer */
    for (int o = 0; o < D3; ++o) d3[o] = (double)W4[o] * dcelu(z3[o]);
    for (int k = 0; k < D2; ++k) {
        double s = 0.0;
        for (int o = 0; o < D3; ++o) s += d3[o] * (double)W3[o * D2 + k];
        d2[k] = s * dcelu(z2[k]);
    }
    for (int k = 0; k < D1; ++k) {
        double s = 0.0;
        for (int o = 0; o < D2; ++o) s += d2[o] * (double)W2[o * D1 + k];
        d1[k] = s * dcelu(z1[k]);
    }
    for (int k = 0; k < AEV_LEN; ++k) {
        double s = 0.0;
        for (int o = 0; o < D1; ++o) s += d1[o] * (double)W1[o * AEV_LEN + k];
        g[k] = s;
    }
}

/* exported pieces for per-stage parity and pins (P1, P2, P5) */
void oracle_aev(int n_atoms, const double *pos, const int32_t *species,
                const int32_t *r_off, const int32_t *r_idx,
                const int32_t *a_off, const int32_t *a_idx, double *aev) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < n_atoms; ++i)
        atom_aev(pos, species, i, r_idx + r_off[i], r_off[i + 1] - r_off[i],
                 a_idx + a_off[i], a_off[i + 1] - a_off[i], aev + (size_t)AEV_LEN * i);
}
void oracle_mlp(int n_rows, const int32_t *species, const double *aev, const float *weights,
                double *e, double *g) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < n_rows; ++i)
        mlp_fwd_bwd(weights + (size_t)W_PER_ELEM * species[i], aev + (size_t)AEV_LEN * i,
                    e + i, g ? g + (size_t)AEV_LEN * i : NULL);
}

/* ---- O7: dE/dx from g_i = dE/daev_i by the chain rule ----------------------
 * Adds the contribution of centre i to grad[N][3] (grad = +dE/dx). */
static void atom_grad(const double *pos, const int32_t *species, int i,
                      const int32_t *rj, int nr, const int32_t *aj, int na,
                      const double *g, double *grad) {
    const double *xi = pos + 3 * i;
    for (int n = 0; n < nr; ++n) {                       /* radial terms */
        int j = rj[n];
        double d[3] = {pos[3 * j] - xi[0], pos[3 * j + 1] - xi[1], pos[3 * j + 2] - xi[2]};
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double fc = fcut(r, RC_R), dfc = dfcut(r, RC_R);
        double dEdr = 0.0;
        for (int k = 0; k < NSHF_R; ++k) {
            double dr = r - (double)SHF_R_F[k];
            double ex = exp(-ETA_R * dr * dr);
            dEdr += g[NSHF_R * species[j] + k] * 0.25 * ex * (-2.0 * ETA_R * dr * fc + dfc);
        }
        for (int c = 0; c < 3; ++c) {                    /* dr/dx_j = u, dr/dx_i = -u */
            double u = d[c] / r;
            grad[3 * j + c] += dEdr * u;
            grad[3 * i + c] -= dEdr * u;
        }
    }
    for (int n = 0; n < na; ++n) {                       /* angular terms */
        int j = aj[n];
        double vj[3] = {pos[3 * j] - xi[0], pos[3 * j + 1] - xi[1], pos[3 * j + 2] - xi[2]};
        double rjn = sqrt(vj[0] * vj[0] + vj[1] * vj[1] + vj[2] * vj[2]);
        double uj[3] = {vj[0] / rjn, vj[1] / rjn, vj[2] / rjn};
        for (int m = n + 1; m < na; ++m) {
            int k = aj[m];
            double vk[3] = {pos[3 * k] - xi[0], pos[3 * k + 1] - xi[1], pos[3 * k + 2] - xi[2]};
            double rkn = sqrt(vk[0] * vk[0] + vk[1] * vk[1] + vk[2] * vk[2]);
            double uk[3] = {vk[0] / rkn, vk[1] / rkn, vk[2] / rkn};
            double cosphi = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
            double c = COS_SCALE * cosphi;
            double theta = acos(c);
            double dtheta_dcosphi = -COS_SCALE / sqrt(1.0 - c * c);
            double rbar = 0.5 * (rjn + rkn);
            double fcj = fcut(rjn, RC_A), fck = fcut(rkn, RC_A);
            double dfcj = dfcut(rjn, RC_A), dfck = dfcut(rkn, RC_A);
            int p = pair_index(species[j], species[k]);
            /* dE/dtheta, dE/drj, dE/drk summed over the 32 terms of this triple */
            double dE_dtheta = 0.0, dE_drj = 0.0, dE_drk = 0.0;
            double A[NSHF_Z], dA[NSHF_Z];                /* same for every a */
            for (int b = 0; b < NSHF_Z; ++b) {
                double x = theta - (double)SHF_Z_F[b];
                double q = 0.5 * (1.0 + cos(x));
                A[b] = pow(q, 32.0);
                dA[b] = -16.0 * pow(q, 31.0) * sin(x);   /* dA/dtheta */
            }
            for (int a = 0; a < NSHF_A; ++a) {
                double dr = rbar - (double)SHF_A_F[a];
                double B = exp(-ETA_A * dr * dr);
                double dB = -2.0 * ETA_A * dr * B;           /* dB/drbar */
                for (int b = 0; b < NSHF_Z; ++b) {
                    double gg = g[RAD_LEN + 32 * p + 8 * a + b];
                    dE_dtheta += gg * 2.0 * dA[b] * B * fcj * fck;
                    dE_drj += gg * 2.0 * A[b] * fck * (0.5 * dB * fcj + B * dfcj);
                    dE_drk += gg * 2.0 * A[b] * fcj * (0.5 * dB * fck + B * dfck);
                }
            }
            double dE_dcos = dE_dtheta * dtheta_dcosphi;
            for (int cc = 0; cc < 3; ++cc) {
                double dcos_dxj = (uk[cc] - cosphi * uj[cc]) / rjn;
                double dcos_dxk = (uj[cc] - cosphi * uk[cc]) / rkn;
                double gj = dE_dcos * dcos_dxj + dE_drj * uj[cc];
                double gk = dE_dcos * dcos_dxk + dE_drk * uk[cc];
                grad[3 * j + cc] += gj;
                grad[3 * k + cc] += gk;
                grad[3 * i + cc] -= gj + gk;
            }
        }
    }
}

/* O1-O7.  pos fp64 [N][3] (lists are decided on (float)pos, O2).  weights fp32
 * (O5 layout).  Outputs: E_sys[n_sys] (O6, index order), F[N][3] = -dE/dx,
 * optional e_atom[N], aev_out[N][384], g_out[N][384].
 * nbr_mode 0 = O(N^2) enumeration (the definition), 1 = cell list (P7-equal). */
int oracle_energy_forces(int n_atoms, int n_sys, const int32_t *sys_off, const double *pos,
                         const int32_t *species, const float *weights, int nbr_mode,
                         double *E_sys, double *F, double *e_atom, double *aev_out, double *g_out) {
    float *posf = (float *)malloc(sizeof(float) * 3 * (size_t)n_atoms);
    for (size_t q = 0; q < 3 * (size_t)n_atoms; ++q) posf[q] = (float)pos[q];
    int32_t *r_off = (int32_t *)malloc(sizeof(int32_t) * ((size_t)n_atoms + 1));
    int32_t *a_off = (int32_t *)malloc(sizeof(int32_t) * ((size_t)n_atoms + 1));
    if (nbr_mode == 0) oracle_neighbors(n_atoms, n_sys, sys_off, posf, r_off, NULL, 0, a_off, NULL, 0);
    else oracle_neighbors_cell(n_atoms, n_sys, sys_off, posf, 5.25, r_off, NULL, 0, a_off, NULL, 0);
    int64_t cr = r_off[n_atoms], ca = a_off[n_atoms];
    int32_t *r_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(cr + 1));
    int32_t *a_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(ca + 1));
    if (nbr_mode == 0) oracle_neighbors(n_atoms, n_sys, sys_off, posf, r_off, r_idx, cr, a_off, a_idx, ca);
    else oracle_neighbors_cell(n_atoms, n_sys, sys_off, posf, 5.25, r_off, r_idx, cr, a_off, a_idx, ca);
    free(posf);

    double *e_loc = (double *)malloc(sizeof(double) * (size_t)n_atoms);
    int nthreads = oracle_num_threads();
    double *grad_t = (double *)calloc((size_t)nthreads * 3 * (size_t)n_atoms, sizeof(double));
#pragma omp parallel
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        double *grad = grad_t + (size_t)tid * 3 * (size_t)n_atoms;
        double aev[AEV_LEN], g[AEV_LEN];
#pragma omp for schedule(dynamic, 8)
        for (int i = 0; i < n_atoms; ++i) {
            const int32_t *rj = r_idx + r_off[i], *aj = a_idx + a_off[i];
            int nr = r_off[i + 1] - r_off[i], na = a_off[i + 1] - a_off[i];
            atom_aev(pos, species, i, rj, nr, aj, na, aev);
            mlp_fwd_bwd(weights + (size_t)W_PER_ELEM * species[i], aev, &e_loc[i], g);
            atom_grad(pos, species, i, rj, nr, aj, na, g, grad);
            if (aev_out) memcpy(aev_out + (size_t)AEV_LEN * i, aev, sizeof(aev));
            if (g_out) memcpy(g_out + (size_t)AEV_LEN * i, g, sizeof(g));
        }
    }
    for (size_t q = 0; q < 3 * (size_t)n_atoms; ++q) {   /* F = -dE/dx, threads in order */
        double s = 0.0;
        for (int t = 0; t < nthreads; ++t) s += grad_t[(size_t)t * 3 * (size_t)n_atoms + q];
        F[q] = -s;
    }
    for (int s = 0; s < n_sys; ++s) {                    /* O6 */
        double acc = 0.0;
        for (int i = sys_off[s]; i < sys_off[s + 1]; ++i) acc += e_loc[i];
        E_sys[s] = acc;
    }
    if (e_atom) memcpy(e_atom, e_loc, sizeof(double) * (size_t)n_atoms);
    free(e_loc); free(grad_t); free(r_off); free(a_off); free(r_idx); free(a_idx);
    return 0;
}

/* P10 test hook: harmonic pair E = k/2 (r01 - r0)^2 between the first two atoms
 * of every system.  Used ONLY to pin the integrator against the textbook
 * oscillator; selected by potential_kind = 1 in oracle_step. */
static void harmonic_energy_forces(int n_sys, const int32_t *sys_off, const double *pos,
                                   double kspring, double r0, double *E_sys, double *F, int n_atoms) {
    memset(F, 0, sizeof(double) * 3 * (size_t)n_atoms);
    for (int s = 0; s < n_sys; ++s) {
        int a = sys_off[s], b = a + 1;
        double d[3] = {pos[3 * b] - pos[3 * a], pos[3 * b + 1] - pos[3 * a + 1], pos[3 * b + 2] - pos[3 * a + 2]};
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        E_sys[s] = 0.5 * kspring * (r - r0) * (r - r0);
        for (int c = 0; c < 3; ++c) {
            double f = -kspring * (r - r0) * d[c] / r;   /* force on b */
            F[3 * b + c] += f;
            F[3 * a + c] -= f;
        }
    }
}

/* O8: velocity-Verlet, fp64.  a = F*ACC/m; v += dt/2 a; x += dt v; F(x);
 * v += dt/2 a.  pos, vel updated in place; F_out = forces at the final
 * positions; pe_hist/ke_hist [(n_steps+1)][n_sys] (eV) record every step
 * including step 0 when non-NULL.  KE = sum m v^2 / (2 ACC). */
int oracle_step(int n_atoms, int n_sys, const int32_t *sys_off, double *pos, double *vel,
                const int32_t *species, const float *weights, const double *masses,
                double dt, int n_steps, int nbr_mode, int potential_kind,
                double kspring, double r0,
                double *F_out, double *pe_hist, double *ke_hist) {
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)n_atoms);
    double *E = (double *)malloc(sizeof(double) * (size_t)n_sys);
#define EVAL()                                                                                   \
    do {                                                                                         \
        if (potential_kind == 1) harmonic_energy_forces(n_sys, sys_off, pos, kspring, r0, E, F, n_atoms); \
        else oracle_energy_forces(n_atoms, n_sys, sys_off, pos, species, weights, nbr_mode, E, F, NULL, NULL, NULL); \
    } while (0)
#define RECORD(step)                                                                             \
    do {                                                                                         \
        for (int s = 0; s < n_sys; ++s) {                                                        \
            double ke = 0.0;                                                                     \
            for (int i = sys_off[s]; i < sys_off[s + 1]; ++i)                                    \
                ke += 0.5 * masses[species[i]] *                                                 \
                      (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]) / ACC; \
            if (pe_hist) pe_hist[(size_t)(step) * n_sys + s] = E[s];                             \
            if (ke_hist) ke_hist[(size_t)(step) * n_sys + s] = ke;                               \
        }                                                                                        \
    } while (0)
    EVAL();
    RECORD(0);
    for (int step = 1; step <= n_steps; ++step) {
        for (int i = 0; i < n_atoms; ++i) {
            double im = ACC / masses[species[i]];
            for (int c = 0; c < 3; ++c) {
                vel[3 * i + c] += 0.5 * dt * F[3 * i + c] * im;
                pos[3 * i + c] += dt * vel[3 * i + c];
            }
        }
        EVAL();
        for (int i = 0; i < n_atoms; ++i) {
            double im = ACC / masses[species[i]];
            for (int c = 0; c < 3; ++c) vel[3 * i + c] += 0.5 * dt * F[3 * i + c] * im;
        }
        RECORD(step);
    }
    if (F_out) memcpy(F_out, F, sizeof(double) * 3 * (size_t)n_atoms);
#undef EVAL
#undef RECORD
    free(F); free(E);
    return 0;
}

/* ---- O9: Langevin dynamics (the paper's timing protocol, PAPER.md:94:
 * "Langevin integrator, friction 0.1 ps^-1").  The paper names no splitting; reading S27 takes
 * BAOAB (Leimkuhler & Matthews) built on the O8 kicks:
 *   B: v += dt/2 a(x)      A: x += dt/2 v
 *   O: v = c1 v + c2 sqrt(kB T ACC / m) xi,  c1 = exp(-gamma dt), c2 = sqrt(1 - c1^2)
 *   A: x += dt/2 v         F(x)         B: v += dt/2 a(x)
 * gamma = 0 gives c1 = 1, c2 = 0: velocity-Verlet.  The normals xi are NOT drawn here from a
 * library stream: both sides implement the same counter-based generator (reading S28):
 * Philox4x32-10 (Salmon et al., SC'11) with counter (atom, step, 0, 0), key (seed_lo, seed_hi);
 * u = ((word >> 8) + 0.5) 2^-24; Box-Muller: xi_x = r cos(2 pi u1), xi_y = r sin(2 pi u1) with
 * r = sqrt(-2 ln u0) from words 0,1; xi_z = sqrt(-2 ln u2) cos(2 pi u3) from words 2,3. */
static const double KB_EV = 8.617333262e-5;      /* eV/K */

static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
void oracle_philox4x32_10(const uint32_t *ctr, const uint32_t *key, uint32_t *out) { philox4x32_10(ctr, key, out); }

/* the three standard normals of (atom, step) */
void oracle_langevin_normals(uint32_t atom, uint32_t step, uint64_t seed, double xi[3]) {
    uint32_t ctr[4] = {atom, step, 0u, 0u}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, w[4];
    philox4x32_10(ctr, key, w);
    double u[4];
    for (int q = 0; q < 4; ++q) u[q] = ((double)(w[q] >> 8) + 0.5) * (1.0 / 16777216.0);
    double r = sqrt(-2.0 * log(u[0]));
    xi[0] = r * cos(2.0 * PI * u[1]);
    xi[1] = r * sin(2.0 * PI * u[1]);
    xi[2] = sqrt(-2.0 * log(u[2])) * cos(2.0 * PI * u[3]);
}

/* n_steps of BAOAB; step indices step0+1 .. step0+n_steps feed the generator.  potential_kind 2 = no
 * forces (free particles: the O step alone thermalises, used by the pins). */
int oracle_step_langevin(int n_atoms, int n_sys, const int32_t *sys_off, double *pos, double *vel,
                         const int32_t *species, const float *weights, const double *masses,
                         double dt, int n_steps, int nbr_mode, int potential_kind,
                         double gamma, double temperature, uint64_t seed, uint32_t step0, double *F_out) {
    double *F = (double *)calloc(3 * (size_t)n_atoms, sizeof(double));
    double *E = (double *)malloc(sizeof(double) * (size_t)n_sys);
    const double c1 = exp(-gamma * dt), c2 = sqrt(1.0 - c1 * c1);
    if (potential_kind == 0)
        oracle_energy_forces(n_atoms, n_sys, sys_off, pos, species, weights, nbr_mode, E, F, NULL, NULL, NULL);
    for (int step = 1; step <= n_steps; ++step) {
        for (int i = 0; i < n_atoms; ++i) {
            double im = ACC / masses[species[i]], xi[3];
            double sigma = sqrt(KB_EV * temperature * im);
            oracle_langevin_normals((uint32_t)i, step0 + (uint32_t)step, seed, xi);
            for (int c = 0; c < 3; ++c) {
                vel[3 * i + c] += 0.5 * dt * F[3 * i + c] * im;          /* B */
                pos[3 * i + c] += 0.5 * dt * vel[3 * i + c];             /* A */
                vel[3 * i + c] = c1 * vel[3 * i + c] + c2 * sigma * xi[c];   /* O */
                pos[3 * i + c] += 0.5 * dt * vel[3 * i + c];             /* A */
            }
        }
        if (potential_kind == 0)
            oracle_energy_forces(n_atoms, n_sys, sys_off, pos, species, weights, nbr_mode, E, F, NULL, NULL, NULL);
        for (int i = 0; i < n_atoms; ++i) {
            double im = ACC / masses[species[i]];
            for (int c = 0; c < 3; ++c) vel[3 * i + c] += 0.5 * dt * F[3 * i + c] * im;   /* B */
        }
    }
    if (F_out) memcpy(F_out, F, sizeof(double) * 3 * (size_t)n_atoms);
    free(F); free(E);
    return 0;
}
