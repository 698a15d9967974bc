/* aims_synth/_heavy.c -- the three loops of the synthetic-input generator that are too slow in numpy.
 *
 * INPUT GENERATION ONLY.  Nothing here is part of the method of arXiv:1912.06636 (no basis evaluation,
 * no culling, no contraction): it makes the *inputs* both the CPU oracle and the CUDA path consume --
 * partition-of-unity integration weights ("partition-of-unity approach ... Stratmann"),
 * the synthetic potential v(r) / GGA vector field g(r), and the cut-plane
 * batching of the point cloud.  Built with gcc by aims_synth/_build.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- cell list over atoms */
typedef struct {
  double lo[3], h;
  int n[3];
  int *start; /* [ncell+1] */
  int *items; /* [n_atoms] */
} cell_list;

static void cl_build(cell_list *cl, int n_atoms, const double *xyz, double h) {
  for (int c = 0; c < 3; c++) {
    double lo = 1e300, hi = -1e300;
    for (int a = 0; a < n_atoms; a++) {
      if (xyz[3 * a + c] < lo) lo = xyz[3 * a + c];
      if (xyz[3 * a + c] > hi) hi = xyz[3 * a + c];
    }
    cl->lo[c] = lo;
    cl->n[c] = (int)floor((hi - lo) / h) + 1;
  }
  cl->h = h;
  int nc = cl->n[0] * cl->n[1] * cl->n[2];
  cl->start = (int *)calloc((size_t)nc + 1, sizeof(int));
  cl->items = (int *)malloc(sizeof(int) * (size_t)(n_atoms > 0 ? n_atoms : 1));
  int *cid = (int *)malloc(sizeof(int) * (size_t)(n_atoms > 0 ? n_atoms : 1));
  for (int a = 0; a < n_atoms; a++) {
    int i[3];
    for (int c = 0; c < 3; c++) {
      i[c] = (int)floor((xyz[3 * a + c] - cl->lo[c]) / h);
      if (i[c] >= cl->n[c]) i[c] = cl->n[c] - 1;
    }
    cid[a] = (i[0] * cl->n[1] + i[1]) * cl->n[2] + i[2];
    cl->start[cid[a] + 1]++;
  }
  for (int k = 0; k < nc; k++) cl->start[k + 1] += cl->start[k];
  int *fill = (int *)calloc((size_t)nc, sizeof(int));
  for (int a = 0; a < n_atoms; a++) cl->items[cl->start[cid[a]] + fill[cid[a]]++] = a; /* ascending a per cell */
  free(fill);
  free(cid);
}
static void cl_free(cell_list *cl) { free(cl->start); free(cl->items); }

/* atoms with |r - R_a| <= rad, ascending atom index; returns count (<= cap) */
static int cl_query(const cell_list *cl, const double *axyz, const double *r, double rad, int *out, double *dout, int cap) {
  int lo[3], hi[3];
  for (int c = 0; c < 3; c++) {
    lo[c] = (int)floor((r[c] - rad - cl->lo[c]) / cl->h);
    hi[c] = (int)floor((r[c] + rad - cl->lo[c]) / cl->h);
    if (lo[c] < 0) lo[c] = 0;
    if (hi[c] >= cl->n[c]) hi[c] = cl->n[c] - 1;
  }
  int m = 0;
  for (int i = lo[0]; i <= hi[0]; i++)
    for (int j = lo[1]; j <= hi[1]; j++)
      for (int k = lo[2]; k <= hi[2]; k++) {
        int c = (i * cl->n[1] + j) * cl->n[2] + k;
        for (int q = cl->start[c]; q < cl->start[c + 1]; q++) {
          int a = cl->items[q];
          double dx = r[0] - axyz[3 * a], dy = r[1] - axyz[3 * a + 1], dz = r[2] - axyz[3 * a + 2];
          double d = sqrt(dx * dx + dy * dy + dz * dz);
          if (d <= rad && m < cap) { out[m] = a; dout[m] = d; m++; }
        }
      }
  /* insertion sort by atom index so the result does not depend on the cell traversal */
  for (int i = 1; i < m; i++) {
    int a = out[i]; double d = dout[i]; int j = i - 1;
    while (j >= 0 && out[j] > a) { out[j + 1] = out[j]; dout[j + 1] = dout[j]; j--; }
    out[j + 1] = a; dout[j + 1] = d;
  }
  return m;
}

/* ---------------------------------------------------------------- Stratmann partition of unity
 * Cell function of Stratmann, Scuseria, Frisch (1996), a = 0.64:
 *   mu_AB = (d_A - d_B)/R_AB, x = clamp(mu/a, -1, 1), z = (35x - 35x^3 + 21x^5 - 5x^7)/16, s = (1 - z)/2,
 *   P_A(r) = prod_{B in cand(r), B != A} s(mu_AB),  w_A(r) = P_A / sum_{B in cand(r)} P_B,
 * cand(r) = atoms within r_part of r ("O(N_atom)" neighbour restriction).  cand depends on r
 * only, so sum_A w_A(r) = 1 for every r.  out[p] = w_{owner[p]}(xyz[p]).  Returns max |cand|, or -1 if cap hit.
 */
static double stratmann_s(double mu) {
  double x = mu / 0.64;
  if (x <= -1.0) return 1.0;
  if (x >= 1.0) return 0.0;
  double x2 = x * x;
  double z = x * (35.0 + x2 * (-35.0 + x2 * (21.0 - 5.0 * x2))) / 16.0;
  double s = 0.5 * (1.0 - z);
  return s < 0.0 ? 0.0 : (s > 1.0 ? 1.0 : s); /* rounding of the polynomial near |x| = 1 */
}

#define CAND_CAP 1024
int synth_partition_weights(int n_atoms, const double *atom_xyz, int64_t n_points, const double *xyz,
                            const int32_t *owner, double r_part, double *w_out) {
  cell_list cl;
  cl_build(&cl, n_atoms, atom_xyz, r_part);
  int worst = 0;
#pragma omp parallel for schedule(dynamic, 2048) reduction(max : worst)
  for (int64_t p = 0; p < n_points; p++) {
    int cand[CAND_CAP];
    double d[CAND_CAP];
    int m = cl_query(&cl, atom_xyz, xyz + 3 * p, r_part, cand, d, CAND_CAP);
    if (m >= CAND_CAP) { worst = 1 << 30; w_out[p] = 0.0; continue; }
    if (m > worst) worst = m;
    int own = owner[p];
    double sum = 0.0, pown = 0.0;
    int inear = 0;
    for (int i = 1; i < m; i++) if (d[i] < d[inear]) inear = i;
    for (int i = 0; i < m; i++) {
      const double *Ra = atom_xyz + 3 * cand[i];
      double P = 1.0;
      /* nearest atom first: it zeroes most far atoms at once */
      if (i != inear) {
        const double *Rb = atom_xyz + 3 * cand[inear];
        double ex = Ra[0] - Rb[0], ey = Ra[1] - Rb[1], ez = Ra[2] - Rb[2];
        P *= stratmann_s((d[i] - d[inear]) / sqrt(ex * ex + ey * ey + ez * ez));
      }
      for (int j = 0; j < m && P != 0.0; j++) {
        if (j == i || j == inear) continue;
        const double *Rb = atom_xyz + 3 * cand[j];
        double ex = Ra[0] - Rb[0], ey = Ra[1] - Rb[1], ez = Ra[2] - Rb[2];
        P *= stratmann_s((d[i] - d[j]) / sqrt(ex * ex + ey * ey + ez * ez));
      }
      sum += P;
      if (cand[i] == own) pown = P;
    }
    w_out[p] = (sum > 0.0) ? pown / sum : 0.0;
  }
  cl_free(&cl);
  return worst >= (1 << 30) ? -1 : worst;
}

/* ---------------------------------------------------------------- smooth synthetic fields (inputs)
 * v(r) = sum_{a: d<r_field} sum_k c[a][k] exp(-alpha[a][k] d^2),  g(r) = sum_{a: d<r_field} b[a] (r-R_a) exp(-beta[a] d^2)
 * g is written as [3][n_points] (component-major) when g != NULL.
 */
int synth_fields(int n_atoms, const double *atom_xyz, int n_gauss, const double *c, const double *alpha,
                 const double *b, const double *beta, double r_field, int64_t n_points, const double *xyz,
                 double *v, double *g) {
  cell_list cl;
  cl_build(&cl, n_atoms, atom_xyz, r_field);
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 2048) reduction(| : bad)
  for (int64_t p = 0; p < n_points; p++) {
    int cand[CAND_CAP];
    double d[CAND_CAP];
    int m = cl_query(&cl, atom_xyz, xyz + 3 * p, r_field, cand, d, CAND_CAP);
    if (m >= CAND_CAP) bad = 1;
    double vs = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    for (int i = 0; i < m; i++) {
      int a = cand[i];
      double d2 = d[i] * d[i];
      for (int k = 0; k < n_gauss; k++) vs += c[a * n_gauss + k] * exp(-alpha[a * n_gauss + k] * d2);
      if (g) {
        double e = b[a] * exp(-beta[a] * d2);
        gx += e * (xyz[3 * p] - atom_xyz[3 * a]);
        gy += e * (xyz[3 * p + 1] - atom_xyz[3 * a + 1]);
        gz += e * (xyz[3 * p + 2] - atom_xyz[3 * a + 2]);
      }
    }
    v[p] = vs;
    if (g) { g[p] = gx; g[n_points + p] = gy; g[2 * n_points + p] = gz; }
  }
  cl_free(&cl);
  return bad ? -1 : 0;
}

/* ---------------------------------------------------------------- cut-plane bisection batching
 * Reading P12 of PAPER.md L210-212 ("grid adapted cut-plane method ... until some targeted number
 * of points per subset is reached"): a set of n points is a batch if n <= max_pts; else with nb = ceil(n/max_pts)
 * the n_left = round(floor(nb/2) * n / nb) points smallest in (coordinate along the axis of largest extent,
 * original index) go left, the rest right; children in depth-first order.  Sizes depend on n only.
 */
typedef struct { double key; int64_t idx; } kv;
static int kv_cmp(const void *a, const void *b) {
  const kv *x = (const kv *)a, *y = (const kv *)b;
  if (x->key < y->key) return -1;
  if (x->key > y->key) return 1;
  return (x->idx > y->idx) - (x->idx < y->idx);
}
static int64_t n_left_of(int64_t n, int max_pts) {
  int64_t nb = (n + max_pts - 1) / max_pts, h = nb / 2;
  return (2 * h * n + nb) / (2 * nb);
}
static void bisect_sizes(int64_t lo, int64_t n, int max_pts, int64_t *ptr, int64_t *nb) {
  if (n <= max_pts) { ptr[(*nb)++] = lo; return; }
  int64_t nl = n_left_of(n, max_pts);
  bisect_sizes(lo, nl, max_pts, ptr, nb);
  bisect_sizes(lo + nl, n - nl, max_pts, ptr, nb);
}
static void bisect_data(const double *xyz, int64_t *order, int64_t n, int max_pts) {
  if (n <= max_pts) return;
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int64_t i = 0; i < n; i++)
    for (int c = 0; c < 3; c++) {
      double x = xyz[3 * order[i] + c];
      if (x < lo[c]) lo[c] = x;
      if (x > hi[c]) hi[c] = x;
    }
  int ax = 0;
  if (hi[1] - lo[1] > hi[ax] - lo[ax]) ax = 1;
  if (hi[2] - lo[2] > hi[ax] - lo[ax]) ax = 2;
  kv *t = (kv *)malloc(sizeof(kv) * (size_t)n);
  for (int64_t i = 0; i < n; i++) { t[i].key = xyz[3 * order[i] + ax]; t[i].idx = order[i]; }
  qsort(t, (size_t)n, sizeof(kv), kv_cmp);
  for (int64_t i = 0; i < n; i++) order[i] = t[i].idx;
  free(t);
  int64_t nl = n_left_of(n, max_pts);
#pragma omp task if (n > 20000)
  bisect_data(xyz, order, nl, max_pts);
#pragma omp task if (n > 20000)
  bisect_data(xyz, order + nl, n - nl, max_pts);
#pragma omp taskwait
}
/* order[n]: out permutation (new position -> original index); batch_ptr: capacity >= 2*ceil(n/max_pts)+2.
 * Returns the number of batches. */
int64_t synth_bisect(int64_t n, const double *xyz, int max_pts, int64_t *order, int64_t *batch_ptr) {
  int64_t nb = 0;
  for (int64_t i = 0; i < n; i++) order[i] = i;
  if (n == 0) { batch_ptr[0] = 0; return 0; }
  bisect_sizes(0, n, max_pts, batch_ptr, &nb);
  batch_ptr[nb] = n;
#pragma omp parallel
#pragma omp single
  bisect_data(xyz, order, n, max_pts);
  return nb;
}
