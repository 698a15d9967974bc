/* oracle/aims_oracle.c -- plain, slow FP64 CPU statement of the real-space grid operations of
 * arXiv:1912.06636 (Huhn, Lange, Yu, Yoon, Blum).  Citations are /root/reference/PAPER.md line numbers.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * constant generator with paper_1912_06636_b200/ (the CUDA path) and neither includes the other.
 *
 * What it computes (the method reaches the plain definition exactly -- it only skips exact zeros -- so the
 * oracle is the definition written out; no blocking, no fusion, no reordering beyond the batch loop the
 * paper itself states):
 *   O1  phi_i(r) = R_s(|r-R_a|) * Y_lm((r-R_a)/|r-R_a|), exactly 0 for |r-R_a|^2 >= rcut^2, and its gradient
 *       (basis functions on grid points: "calculate_phi", Fig. 6 L322/L356; L314; cutoff L202).
 *   O2  nnz(B) = functions "that are nonzero on at least part of the grid points in this batch" (L235).
 *   O3  h_ij[B] = sum_{r in B} w(r) phi_i(r) (h phi_j)(r)   (Eq. 24, Eq. 25-27), h = sum_B h[B]
 *       (Eq. 23), with h_KS -> local potential v(r) plus the GGA term in its integrated-by-parts form
 *       sum_r w g.(grad phi_i phi_j + phi_i grad phi_j) (L67; Eq. 18; reading P2).
 *       Overlap s_ij: same with v = 1, g absent (Eq. 5 "exactly analogous").
 *   O4  n(r) = sum_ij phi_i(r) n_ij phi_j(r) (Eq. 3) restricted to nnz(B) (L235, L314 "reduction of the
 *       density matrix ... to the dense-but-smaller n_ij"), computed as temp = n_ij phi, n = temp . phi
 *       (Fig. 6b); grad n = 2 sum_ij grad phi_i n_ij phi_j for symmetric n_ij (L67, L93-95).
 *   O5  Pulay forces F_at (Eq. 16 and Eq. 18) for the reduced h_KS; see the block at the end of this file.
 *   O6+ (blocks further down, each with its own header and pins): kinetic term of h_KS and the meta-GGA tau matrix
 *       (Eq. 26, Fig. 6a), Hessian of the density (L93-95), Bloch sums for periodic systems (Eq. 7, 11, 12), the
 *       Stratmann partition of unity (Eq. 21-22, reading P5).
 *
 * Pins (tests/test_oracle_pins.py): Y_lm vs scipy and orthonormality by exact product quadrature; spline vs
 * scipy CubicSpline; grad phi vs finite differences; Gaussian overlap closed form; S symmetric PSD;
 * sum_p w n = Tr(D S), sum_p w v n = Tr(D H_LDA), sum_p w g.grad n = Tr(D H_GGA); batched == brute force;
 * invariance under re-batching; Hessian of phi vs finite differences of grad phi; Pulay forces vs central differences
 * of Tr(D H(R)) - Tr(Q S(R)) under atom displacement and vs the term-by-term brute force.  The paper prints no numerical value for this path, so no pin is "the paper's
 * number"; all pins are mathematical.
 *
 * Arithmetic: IEEE double, no FMA contraction (built with -ffp-contract=off), sums in the loop order written.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  /* basis */
  int32_t n_atoms, n_species, n_shells, n_splines, n_knots;
  const double *atom_xyz;           /* [n_atoms][3] */
  const int32_t *atom_species;      /* [n_atoms] */
  const int32_t *species_shell_ptr; /* [n_species+1] */
  const int32_t *shell_l;           /* [n_shells] */
  const double *shell_rcut;         /* [n_shells] */
  const int32_t *shell_spline;      /* [n_shells] */
  double r0, log_inc;
  const double *spline_coef;        /* [n_splines][n_knots-1][4] */
  /* grid */
  int64_t n_points;
  int32_t n_batches;
  const double *xyz;                /* [n_points][3] */
  const double *w;                  /* [n_points] */
  const int64_t *batch_ptr;         /* [n_batches+1] */
  /* atom-pair block pattern, upper blocks */
  const int64_t *row_ptr;           /* [n_atoms+1] */
  const int32_t *col_atom;          /* [n_blocks] */
  const int64_t *blk_off;           /* [n_blocks] */
  const int32_t *blk_ld;            /* [n_blocks] */
  int64_t n_values;
} orc_system;

/* number of OpenMP threads the batch loops use (reported by bench.py's cpu_baseline; no arithmetic) */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif

/* ------------------------------------------------------------------ real spherical harmonics (reading P10)
 * S_lm: homogeneous polynomial of degree l with S_lm(u) = Y_lm(u) on the unit sphere; orthonormal real harmonics,
 * m = -l..l, no Condon-Shortley phase.  Y[m+l]; if gS != NULL also gS[m+l][3] = grad S_lm at (x,y,z). */
void orc_solid_harmonics(int l, const double u[3], double *Y, double (*gS)[3]) {
  const double pi = 3.14159265358979323846;
  double x = u[0], y = u[1], z = u[2];
  if (l == 0) {
    Y[0] = 0.5 * sqrt(1.0 / pi);
    if (gS) { gS[0][0] = 0; gS[0][1] = 0; gS[0][2] = 0; }
  } else if (l == 1) {
    double c = sqrt(3.0 / (4.0 * pi));
    Y[0] = c * y; Y[1] = c * z; Y[2] = c * x;
    if (gS) {
      gS[0][0] = 0; gS[0][1] = c; gS[0][2] = 0;
      gS[1][0] = 0; gS[1][1] = 0; gS[1][2] = c;
      gS[2][0] = c; gS[2][1] = 0; gS[2][2] = 0;
    }
  } else if (l == 2) {
    double a = 0.5 * sqrt(15.0 / pi), b = 0.25 * sqrt(5.0 / pi), c = 0.25 * sqrt(15.0 / pi);
    Y[0] = a * x * y;
    Y[1] = a * y * z;
    Y[2] = b * (2.0 * z * z - x * x - y * y);
    Y[3] = a * x * z;
    Y[4] = c * (x * x - y * y);
    if (gS) {
      gS[0][0] = a * y;        gS[0][1] = a * x;        gS[0][2] = 0;
      gS[1][0] = 0;            gS[1][1] = a * z;        gS[1][2] = a * y;
      gS[2][0] = -2.0 * b * x; gS[2][1] = -2.0 * b * y; gS[2][2] = 4.0 * b * z;
      gS[3][0] = a * z;        gS[3][1] = 0;            gS[3][2] = a * x;
      gS[4][0] = 2.0 * c * x;  gS[4][1] = -2.0 * c * y; gS[4][2] = 0;
    }
  } else if (l == 3) {
    double a = 0.25 * sqrt(35.0 / (2.0 * pi)), b = 0.5 * sqrt(105.0 / pi), c = 0.25 * sqrt(21.0 / (2.0 * pi));
    double d = 0.25 * sqrt(7.0 / pi), e = 0.25 * sqrt(105.0 / pi);
    double x2 = x * x, y2 = y * y, z2 = z * z;
    Y[0] = a * y * (3.0 * x2 - y2);
    Y[1] = b * x * y * z;
    Y[2] = c * y * (4.0 * z2 - x2 - y2);
    Y[3] = d * z * (2.0 * z2 - 3.0 * x2 - 3.0 * y2);
    Y[4] = c * x * (4.0 * z2 - x2 - y2);
    Y[5] = e * z * (x2 - y2);
    Y[6] = a * x * (x2 - 3.0 * y2);
    if (gS) {
      gS[0][0] = a * 6.0 * x * y;            gS[0][1] = a * (3.0 * x2 - 3.0 * y2);      gS[0][2] = 0;
      gS[1][0] = b * y * z;                  gS[1][1] = b * x * z;                      gS[1][2] = b * x * y;
      gS[2][0] = c * (-2.0 * x * y);         gS[2][1] = c * (4.0 * z2 - x2 - 3.0 * y2); gS[2][2] = c * 8.0 * y * z;
      gS[3][0] = d * (-6.0 * x * z);         gS[3][1] = d * (-6.0 * y * z);             gS[3][2] = d * (6.0 * z2 - 3.0 * x2 - 3.0 * y2);
      gS[4][0] = c * (4.0 * z2 - 3.0 * x2 - y2); gS[4][1] = c * (-2.0 * x * y);         gS[4][2] = c * 8.0 * x * z;
      gS[5][0] = e * 2.0 * x * z;            gS[5][1] = e * (-2.0 * y * z);             gS[5][2] = e * (x2 - y2);
      gS[6][0] = a * (3.0 * x2 - 3.0 * y2);  gS[6][1] = a * (-6.0 * x * y);             gS[6][2] = 0;
    }
  }
}

/* ------------------------------------------------------------------ radial function (readings P8, P11)
 * R is *defined* as the tabulated cubic spline in the log-index coordinate:
 *   t = ln(max(d,r0)/r0)/log_inc, k = min(floor(t), n_knots-2), x = t-k, R = a + x(b + x(c + x d)),
 *   dR/dd = (b + 2 c x + 3 d x^2) / (log_inc * max(d,r0)). */
void orc_radial(const orc_system *S, int spline, double d, double *R, double *dR) {
  double dd = d > S->r0 ? d : S->r0;
  double t = log(dd / S->r0) / S->log_inc;
  int k = (int)floor(t);
  if (k > S->n_knots - 2) k = S->n_knots - 2;
  if (k < 0) k = 0;
  double x = t - (double)k;
  const double *c = S->spline_coef + ((size_t)spline * (size_t)(S->n_knots - 1) + (size_t)k) * 4;
  *R = c[0] + x * (c[1] + x * (c[2] + x * c[3]));
  *dR = (c[1] + x * (2.0 * c[2] + x * 3.0 * c[3])) / (S->log_inc * dd);
}

/* squared distance in the pinned operation order of reading P6: ((dx*dx + dy*dy) + dz*dz), separate roundings */
static double dist2(const double *r, const double *Ra, double dv[3]) {
  dv[0] = r[0] - Ra[0]; dv[1] = r[1] - Ra[1]; dv[2] = r[2] - Ra[2];
  double xx = dv[0] * dv[0], yy = dv[1] * dv[1], zz = dv[2] * dv[2];
  double s = xx + yy;
  return s + zz;
}

/* O1: all 2l+1 functions of (atom, shell) at point r: phi[m+l], and if grad != NULL grad[m+l][3].
 * grad phi = (R' - l R/d) Y u + (R/d) grad S_lm(u)   (phi = R(d) S_lm(dvec)/d^l). */
void orc_shell_at_point(const orc_system *S, int atom, int shell, const double r[3], double *phi, double (*grad)[3]) {
  int l = S->shell_l[shell];
  double rc = S->shell_rcut[shell];
  double rc2 = rc * rc;
  double dv[3];
  double d2 = dist2(r, S->atom_xyz + 3 * atom, dv);
  if (!(d2 < rc2)) {
    for (int m = 0; m < 2 * l + 1; m++) {
      phi[m] = 0.0;
      if (grad) { grad[m][0] = 0.0; grad[m][1] = 0.0; grad[m][2] = 0.0; }
    }
    return;
  }
  double d = sqrt(d2);
  double u[3] = {0.0, 0.0, 1.0};                       /* d == 0: direction undefined, take z (P11) */
  if (d > 0.0) { u[0] = dv[0] / d; u[1] = dv[1] / d; u[2] = dv[2] / d; }
  double dd = d > S->r0 ? d : S->r0;
  double R, dR, Y[7], gS[7][3];
  orc_radial(S, S->shell_spline[shell], d, &R, &dR);
  orc_solid_harmonics(l, u, Y, grad ? gS : NULL);
  for (int m = 0; m < 2 * l + 1; m++) {
    phi[m] = R * Y[m];
    if (grad) {
      double f = (dR - (double)l * R / dd) * Y[m];
      for (int c = 0; c < 3; c++) grad[m][c] = f * u[c] + (R / dd) * gS[m][c];
    }
  }
}

/* ------------------------------------------------------------------ global basis index (reading P7)
 * atom-major, then the species' shells in order, then m = -l..l. */
static int atom_n_fn(const orc_system *S, int a) {
  int sp = S->atom_species[a], n = 0;
  for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) n += 2 * S->shell_l[s] + 1;
  return n;
}
/* atom_fn_ptr[n_atoms+1] */
void orc_atom_fn_ptr(const orc_system *S, int64_t *ptr) {
  ptr[0] = 0;
  for (int a = 0; a < S->n_atoms; a++) ptr[a + 1] = ptr[a] + atom_n_fn(S, a);
}
/* offset of block (A,B), A <= B, in the value array and its leading dimension; -1 if the pair is not in the pattern */
static int64_t find_block(const orc_system *S, int A, int B, int *ld) {
  for (int64_t q = S->row_ptr[A]; q < S->row_ptr[A + 1]; q++)
    if (S->col_atom[q] == B) { *ld = S->blk_ld[q]; return S->blk_off[q]; }
  return -1;
}

/* ------------------------------------------------------------------ O2: nnz(B) (L235; reading P6)
 * Function i = (a, s, m) is in nnz(B) iff some point p of B has d2(p,a) < rcut_s^2 (strict); decided per shell.
 * fn_index (capacity: total number of functions) receives the ascending global indices; fn_atom / fn_shell / fn_m
 * (optional, same capacity) the decomposition of each listed function.  Returns |nnz(B)|. */
int orc_batch_nnz(const orc_system *S, int b, int32_t *fn_index, int32_t *fn_atom, int32_t *fn_shell, int32_t *fn_m) {
  int n = 0;
  int64_t g = 0; /* global index of the first function of the current shell */
  for (int a = 0; a < S->n_atoms; a++) {
    int sp = S->atom_species[a];
    for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
      int l = S->shell_l[s];
      double rc2 = S->shell_rcut[s] * S->shell_rcut[s];
      int touches = 0;
      for (int64_t p = S->batch_ptr[b]; p < S->batch_ptr[b + 1] && !touches; p++) {
        double dv[3];
        if (dist2(S->xyz + 3 * p, S->atom_xyz + 3 * a, dv) < rc2) touches = 1;
      }
      if (touches)
        for (int m = -l; m <= l; m++) {
          fn_index[n] = (int32_t)(g + m + l);
          if (fn_atom) fn_atom[n] = a;
          if (fn_shell) fn_shell[n] = s;
          if (fn_m) fn_m[n] = m;
          n++;
        }
      g += 2 * l + 1;
    }
  }
  return n;
}

/* ------------------------------------------------------------------ O1 on a batch ("calculate_phi", L322/L356)
 * phi[i][p] for i in nnz(B) (row-major, n_p = batch size), dphi[c][i][p] if want_grad.  nnz lists as returned by
 * orc_batch_nnz. */
void orc_eval_basis(const orc_system *S, int b, int want_grad, int nnz, const int32_t *fn_atom, const int32_t *fn_shell,
                    const int32_t *fn_m, double *phi, double *dphi) {
  int64_t p0 = S->batch_ptr[b];
  int np = (int)(S->batch_ptr[b + 1] - p0);
  for (int i = 0; i < nnz;) {                         /* the list holds whole shells: rows i .. i+2l of one (atom, shell) */
    int l = S->shell_l[fn_shell[i]];
    for (int p = 0; p < np; p++) {
      double val[7], gr[7][3];
      orc_shell_at_point(S, fn_atom[i], fn_shell[i], S->xyz + 3 * (p0 + p), val, want_grad ? gr : NULL);
      for (int m = 0; m < 2 * l + 1; m++) {
        phi[(size_t)(i + m) * np + p] = val[m];
        if (want_grad)
          for (int c = 0; c < 3; c++) dphi[((size_t)c * nnz + i + m) * np + p] = gr[m][c];
      }
    }
    i += 2 * l + 1;
  }
  (void)fn_m;
}

/* ------------------------------------------------------------------ O3: Hamiltonian / overlap integration
 * For every listed batch B: h_ij[B] = sum_{p in B} w_p phi_i v_p phi_j                     (Eq. 24-27)
 *                                   + sum_{p in B} w_p [ (g_p.grad phi_i) phi_j + phi_i (g_p.grad phi_j) ]   (P2)
 * for i, j in nnz(B); added into H_values (Eq. 23; "insert_into_h", L327) for atom pairs in the upper pattern
 * (diagonal atom blocks hold the full square).  g == NULL: LDA.  H_values is accumulated into (caller zeroes). */
void orc_integrate_hamiltonian(const orc_system *S, int n_sel, const int32_t *batches, const double *v, const double *g,
                               double *H_values) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (nnz == 0 || np == 0) continue;
    double *phi = (double *)malloc(sizeof(double) * (size_t)nnz * np * (g ? 4 : 1));
    double *dphi = g ? phi + (size_t)nnz * np : NULL;
    orc_eval_basis(S, b, g != NULL, nnz, fa, fs, fm, phi, dphi);
    /* G_ip = g_p . grad phi_i(r_p) */
    double *G = NULL;
    if (g) {
      G = (double *)malloc(sizeof(double) * (size_t)nnz * np);
      for (int i = 0; i < nnz; i++)
        for (int p = 0; p < np; p++) {
          double s = 0.0;
          for (int c = 0; c < 3; c++) s += g[(size_t)c * S->n_points + p0 + p] * dphi[((size_t)c * nnz + i) * np + p];
          G[(size_t)i * np + p] = s;
        }
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nnz; i++) {
      int A = fa[i];
      int ai = (int)(idx[i] - afp[A]);
      for (int j = 0; j < nnz; j++) {
        int B = fa[j];
        if (B < A) continue;                         /* lower atom blocks are not stored */
        int ld;
        int64_t off = find_block(S, A, B, &ld);
        if (off < 0) continue;                       /* pair outside the pattern: the product is identically zero */
        int bj = (int)(idx[j] - afp[B]);
        double h = 0.0;
        for (int p = 0; p < np; p++) {
          double wp = S->w[p0 + p];
          double pi_ = phi[(size_t)i * np + p], pj = phi[(size_t)j * np + p];
          double term = wp * pi_ * v[p0 + p] * pj;
          if (g) term += wp * (G[(size_t)i * np + p] * pj + pi_ * G[(size_t)j * np + p]);
          h += term;
        }
        H_values[off + (int64_t)ai * ld + bj] += h;
      }
    }
    free(G);
    free(phi);
  }
  free(idx);
  free(afp);
}

/* ------------------------------------------------------------------ O4: density update
 * For every listed batch B and p in B: n_p = sum_i phi_ip temp_ip, temp_ip = sum_j n_ij[B] phi_jp  (Fig. 6b),
 * n_ij[B] = D restricted to nnz(B) ("calculate_density_mat", L314/L357; zero outside the pattern);
 * grad_n[c][p] = 2 sum_i dphi[c]_ip temp_ip (D symmetric).  Only points of the listed batches are written. */
void orc_update_density(const orc_system *S, int n_sel, const int32_t *batches, const double *D_values, double *n,
                        double *grad_n) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (np == 0) continue;
    double *phi = (double *)malloc(sizeof(double) * ((size_t)nnz * np * (grad_n ? 4 : 1) + 1));
    double *dphi = grad_n ? phi + (size_t)nnz * np : NULL;
    orc_eval_basis(S, b, grad_n != NULL, nnz, fa, fs, fm, phi, dphi);
    /* calculate_density_mat: dense D_b[i][j] */
    double *Db = (double *)malloc(sizeof(double) * ((size_t)nnz * nnz + 1));
    for (int i = 0; i < nnz; i++)
      for (int j = 0; j < nnz; j++) {
        int A = fa[i], B = fa[j];
        int ai = (int)(idx[i] - afp[A]), bj = (int)(idx[j] - afp[B]);
        int ld;
        double val = 0.0;
        if (A <= B) { int64_t off = find_block(S, A, B, &ld); if (off >= 0) val = D_values[off + (int64_t)ai * ld + bj]; }
        else        { int64_t off = find_block(S, B, A, &ld); if (off >= 0) val = D_values[off + (int64_t)bj * ld + ai]; }
        Db[(size_t)i * nnz + j] = val;
      }
#pragma omp parallel for schedule(static)
    for (int p = 0; p < np; p++) {
      double acc = 0.0, gacc[3] = {0.0, 0.0, 0.0};
      for (int i = 0; i < nnz; i++) {
        double t = 0.0;
        for (int j = 0; j < nnz; j++) t += Db[(size_t)i * nnz + j] * phi[(size_t)j * np + p];
        acc += phi[(size_t)i * np + p] * t;
        if (grad_n)
          for (int c = 0; c < 3; c++) gacc[c] += dphi[((size_t)c * nnz + i) * np + p] * t;
      }
      n[p0 + p] = acc;
      if (grad_n)
        for (int c = 0; c < 3; c++) grad_n[(size_t)c * S->n_points + p0 + p] = 2.0 * gacc[c];
    }
    free(Db);
    free(phi);
  }
  free(idx);
  free(afp);
}

/* ------------------------------------------------------------------ brute force (tiny inputs only)
 * No batches, no culling, no block pattern: every function against every function at every point.
 *   Hd[i][j] = sum_p w_p phi_i v_p phi_j + sum_p w_p [(g.grad phi_i) phi_j + phi_i (g.grad phi_j)]   (Eq. 21)
 *   n_p = sum_ij phi_i Dd[i][j] phi_j ,  grad n_p = sum_ij (grad phi_i phi_j + phi_i grad phi_j) Dd[i][j] (Eq. 3)
 * Hd, Dd: dense [n_basis][n_basis].  grad n is written from the product rule, not from the "2 x" shortcut. */
void orc_brute(const orc_system *S, const double *v, const double *g, double *Hd, const double *Dd, double *n,
               double *grad_n) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nb = (int)afp[S->n_atoms];
  double *phi = (double *)malloc(sizeof(double) * (size_t)nb * 4);
  double *dph = phi + nb;                              /* dph[c*nb + i] */
  if (Hd) memset(Hd, 0, sizeof(double) * (size_t)nb * nb);
  for (int64_t p = 0; p < S->n_points; p++) {
    int i = 0;
    for (int a = 0; a < S->n_atoms; a++) {
      int sp = S->atom_species[a];
      for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
        int l = S->shell_l[s];
        double val[7], gr[7][3];
        orc_shell_at_point(S, a, s, S->xyz + 3 * p, val, gr);
        for (int m = 0; m < 2 * l + 1; m++, i++) {
          phi[i] = val[m];
          for (int c = 0; c < 3; c++) dph[c * nb + i] = gr[m][c];
        }
      }
    }
    if (Hd) {
      double wp = S->w[p];
      for (int a = 0; a < nb; a++)
        for (int b = 0; b < nb; b++) {
          double t = wp * phi[a] * v[p] * phi[b];
          if (g)
            for (int c = 0; c < 3; c++)
              t += wp * g[(size_t)c * S->n_points + p] * (dph[c * nb + a] * phi[b] + phi[a] * dph[c * nb + b]);
          Hd[(size_t)a * nb + b] += t;
        }
    }
    if (Dd && n) {
      double acc = 0.0, ga[3] = {0, 0, 0};
      for (int a = 0; a < nb; a++)
        for (int b = 0; b < nb; b++) {
          double dab = Dd[(size_t)a * nb + b];
          acc += phi[a] * dab * phi[b];
          if (grad_n)
            for (int c = 0; c < 3; c++) ga[c] += (dph[c * nb + a] * phi[b] + phi[a] * dph[c * nb + b]) * dab;
        }
      n[p] = acc;
      if (grad_n)
        for (int c = 0; c < 3; c++) grad_n[(size_t)c * S->n_points + p] = ga[c];
    }
  }
  free(phi);
  free(afp);
}

/* ====================================================================================================================
 * Pulay forces (Eq. 14-18; evaluated "alongside the density update"
 * on the same batches, L301-308, L405).  With the reduced h_KS of this build (local potential v plus the GGA term of
 * reading P2, g = 2 df/d|grad n|^2 grad n supplied as a field) and nabla_at phi_i = -grad phi_i for i centred on atom
 * `at`, 0 otherwise, Eq. 16 and Eq. 18 read on the grid
 *   F_at = 2 sum_p w_p sum_{i on at} sum_j { grad phi_i [ n_ij (v_p phi_j + g_p.grad phi_j) - q_ij phi_j ]
 *                                            + (Hess phi_i g_p) n_ij phi_j }                                  (all at r_p)
 * i.e. F_at = -d/dR_at [ Tr(n h(R)) - Tr(q s(R)) ] at fixed n_ij, q_ij, v, g, w and grid -- the pin used in
 * tests/test_oracle_pins.py (central differences of the already pinned H and S).  The atomic-ZORA term (Eq. 19) and
 * the Hellmann-Feynman force (L403, not on this path in the paper either) are outside the reduced h_KS.
 * kinetic != 0: h_KS phi_j in the first term of Eq. 16 also carries -1/2 lap phi_j (row f2), i.e. v_p phi_j -> v_p phi_j - 1/2 lap phi_j.
 * Eq. 16 uses the Hermiticity of h_KS, which holds on the grid only to quadrature accuracy for the kinetic operator, so that
 * part equals -d/dR_at Tr(n t(R)) to grid accuracy only (pinned so), while batched == brute force stays exact.
 * ==================================================================================================================== */

/* second derivatives of the solid harmonics S_lm at (x,y,z): hS[m+l][6] = (xx, yy, zz, xy, xz, yz) */
void orc_solid_harmonics_hess(int l, const double u[3], double (*hS)[6]) {
  const double pi = 3.14159265358979323846;
  double x = u[0], y = u[1], z = u[2];
  for (int m = 0; m < 2 * l + 1; m++)
    for (int k = 0; k < 6; k++) hS[m][k] = 0.0;
  if (l == 2) {
    double a = 0.5 * sqrt(15.0 / pi), b = 0.25 * sqrt(5.0 / pi), c = 0.25 * sqrt(15.0 / pi);
    hS[0][3] = a;                                             /* a x y */
    hS[1][5] = a;                                             /* a y z */
    hS[2][0] = -2.0 * b; hS[2][1] = -2.0 * b; hS[2][2] = 4.0 * b;   /* b (2 z^2 - x^2 - y^2) */
    hS[3][4] = a;                                             /* a x z */
    hS[4][0] = 2.0 * c; hS[4][1] = -2.0 * c;                  /* c (x^2 - y^2) */
  } else if (l == 3) {
    double a = 0.25 * sqrt(35.0 / (2.0 * pi)), b = 0.5 * sqrt(105.0 / pi), c = 0.25 * sqrt(21.0 / (2.0 * pi));
    double d = 0.25 * sqrt(7.0 / pi), e = 0.25 * sqrt(105.0 / pi);
    /* a (3 x^2 y - y^3) */
    hS[0][0] = 6.0 * a * y; hS[0][1] = -6.0 * a * y; hS[0][3] = 6.0 * a * x;
    /* b x y z */
    hS[1][3] = b * z; hS[1][4] = b * y; hS[1][5] = b * x;
    /* c (4 y z^2 - x^2 y - y^3) */
    hS[2][0] = -2.0 * c * y; hS[2][1] = -6.0 * c * y; hS[2][2] = 8.0 * c * y; hS[2][3] = -2.0 * c * x; hS[2][5] = 8.0 * c * z;
    /* d (2 z^3 - 3 x^2 z - 3 y^2 z) */
    hS[3][0] = -6.0 * d * z; hS[3][1] = -6.0 * d * z; hS[3][2] = 12.0 * d * z; hS[3][4] = -6.0 * d * x; hS[3][5] = -6.0 * d * y;
    /* c (4 x z^2 - x^3 - x y^2) */
    hS[4][0] = -6.0 * c * x; hS[4][1] = -2.0 * c * x; hS[4][2] = 8.0 * c * x; hS[4][3] = -2.0 * c * y; hS[4][4] = 8.0 * c * z;
    /* e (x^2 z - y^2 z) */
    hS[5][0] = 2.0 * e * z; hS[5][1] = -2.0 * e * z; hS[5][4] = 2.0 * e * x; hS[5][5] = -2.0 * e * y;
    /* a (x^3 - 3 x y^2) */
    hS[6][0] = 6.0 * a * x; hS[6][1] = -6.0 * a * x; hS[6][3] = -6.0 * a * y;
  }
}

/* radial spline with second derivative: with s = log_inc * max(d,r0),
 *   R' = R_t / s,  R'' = R_tt / s^2 - R_t / (s * max(d,r0)),  R_t = b + 2cx + 3dx^2,  R_tt = 2c + 6dx. */
void orc_radial2(const orc_system *S, int spline, double d, double *R, double *dR, double *d2R) {
  double dd = d > S->r0 ? d : S->r0;
  double t = log(dd / S->r0) / S->log_inc;
  int k = (int)floor(t);
  if (k > S->n_knots - 2) k = S->n_knots - 2;
  if (k < 0) k = 0;
  double x = t - (double)k;
  const double *c = S->spline_coef + ((size_t)spline * (size_t)(S->n_knots - 1) + (size_t)k) * 4;
  double Rt = c[1] + x * (2.0 * c[2] + x * 3.0 * c[3]);
  double Rtt = 2.0 * c[2] + 6.0 * c[3] * x;
  double s = S->log_inc * dd;
  *R = c[0] + x * (c[1] + x * (c[2] + x * c[3]));
  *dR = Rt / s;
  *d2R = Rtt / (s * s) - Rt / (s * dd);
}

/* phi, grad phi and the Hessian hess[m+l][6] = (xx, yy, zz, xy, xz, yz) of the 2l+1 functions of (atom, shell) at r.
 * With phi = F(d) S_lm(dvec), F = R d^-l:
 *   d_c d_e phi = A u_c u_e Y + B (delta_ce - u_c u_e) Y + B (u_c gS_e + u_e gS_c) + (R/d^2) hS_ce,
 *   A = R'' - 2 l R'/d + l(l+1) R/d^2,   B = (R' - l R/d)/d,   Y, gS, hS = S_lm and its derivatives at the unit vector u. */
void orc_shell_hess_at_point(const orc_system *S, int atom, int shell, const double r[3], double *phi, double (*grad)[3],
                             double (*hess)[6]) {
  static const int ic[6] = {0, 1, 2, 0, 0, 1}, ie[6] = {0, 1, 2, 1, 2, 2};
  int l = S->shell_l[shell];
  double rc = S->shell_rcut[shell];
  double rc2 = rc * rc;
  double dv[3];
  double d2 = dist2(r, S->atom_xyz + 3 * atom, dv);
  if (!(d2 < rc2)) {
    for (int m = 0; m < 2 * l + 1; m++) {
      phi[m] = 0.0;
      for (int c = 0; c < 3; c++) grad[m][c] = 0.0;
      for (int k = 0; k < 6; k++) hess[m][k] = 0.0;
    }
    return;
  }
  double d = sqrt(d2);
  double u[3] = {0.0, 0.0, 1.0};
  if (d > 0.0) { u[0] = dv[0] / d; u[1] = dv[1] / d; u[2] = dv[2] / d; }
  double dd = d > S->r0 ? d : S->r0;
  double R, dR, d2R, Y[7], gS[7][3], hS[7][6];
  orc_radial2(S, S->shell_spline[shell], d, &R, &dR, &d2R);
  orc_solid_harmonics(l, u, Y, gS);
  orc_solid_harmonics_hess(l, u, hS);
  double A = d2R - 2.0 * l * dR / dd + (double)(l * (l + 1)) * R / (dd * dd);
  double B = (dR - (double)l * R / dd) / dd;
  for (int m = 0; m < 2 * l + 1; m++) {
    phi[m] = R * Y[m];
    for (int c = 0; c < 3; c++) grad[m][c] = (dR - (double)l * R / dd) * Y[m] * u[c] + (R / dd) * gS[m][c];
    for (int k = 0; k < 6; k++) {
      int c = ic[k], e = ie[k];
      double delta = (c == e) ? 1.0 : 0.0;
      hess[m][k] = A * u[c] * u[e] * Y[m] + B * (delta - u[c] * u[e]) * Y[m] + B * (u[c] * gS[m][e] + u[e] * gS[m][c]) +
                   (R / (dd * dd)) * hS[m][k];
    }
  }
}

/* dense restriction of a block-sparse symmetric matrix to nnz(B) ("calculate_density_mat", L314/L357) */
static void restrict_matrix(const orc_system *S, const int64_t *afp, int nnz, const int32_t *idx, const int32_t *fa,
                            const double *values, double *Mb) {
  for (int i = 0; i < nnz; i++)
    for (int j = 0; j < nnz; j++) {
      int A = fa[i], B = fa[j];
      int ai = (int)(idx[i] - afp[A]), bj = (int)(idx[j] - afp[B]);
      int ld;
      double val = 0.0;
      if (A <= B) { int64_t off = find_block(S, A, B, &ld); if (off >= 0) val = values[off + (int64_t)ai * ld + bj]; }
      else        { int64_t off = find_block(S, B, A, &ld); if (off >= 0) val = values[off + (int64_t)bj * ld + ai]; }
      Mb[(size_t)i * nnz + j] = val;
    }
}

/* Pulay forces on the listed batches, added into F[n_atoms][3] (caller zeroes).  g == NULL: no GGA term;
 * Q_values == NULL: no energy-weighted term.  Per batch: temp matrices  Tn = n_ij phi,  Tg = n_ij (g.grad phi),
 * Tq = q_ij phi  (the DSYMM-shaped products of Fig. 6b), then the point sums of the header formula. */
void orc_pulay_forces(const orc_system *S, int n_sel, const int32_t *batches, const double *v, const double *g,
                      const double *D_values, const double *Q_values, int kinetic, double *F) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (nnz == 0 || np == 0) continue;
    size_t sz = (size_t)nnz * np;
    double *phi = (double *)malloc(sizeof(double) * sz * 10);     /* phi, dphi[3], hess[6] */
    double *dphi = phi + sz, *hes = phi + 4 * sz;
    for (int i = 0; i < nnz;) {
      int l = S->shell_l[fs[i]];
      for (int p = 0; p < np; p++) {
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, fa[i], fs[i], S->xyz + 3 * (p0 + p), val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++) {
          phi[(size_t)(i + m) * np + p] = val[m];
          for (int c = 0; c < 3; c++) dphi[((size_t)c * nnz + i + m) * np + p] = gr[m][c];
          for (int k = 0; k < 6; k++) hes[((size_t)k * nnz + i + m) * np + p] = hh[m][k];
        }
      }
      i += 2 * l + 1;
    }
    double *Db = (double *)malloc(sizeof(double) * (size_t)nnz * nnz);
    double *Qb = Q_values ? (double *)malloc(sizeof(double) * (size_t)nnz * nnz) : NULL;
    restrict_matrix(S, afp, nnz, idx, fa, D_values, Db);
    if (Qb) restrict_matrix(S, afp, nnz, idx, fa, Q_values, Qb);
    double *Frow = (double *)calloc((size_t)nnz * 3, sizeof(double));     /* per-function contribution, summed per atom below */
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nnz; i++) {
      double f[3] = {0.0, 0.0, 0.0};
      for (int p = 0; p < np; p++) {
        double gp[3] = {0.0, 0.0, 0.0};
        if (g) for (int c = 0; c < 3; c++) gp[c] = g[(size_t)c * S->n_points + p0 + p];
        double tn = 0.0, tg = 0.0, tq = 0.0, tk = 0.0;
        for (int j = 0; j < nnz; j++) {
          double dij = Db[(size_t)i * nnz + j];
          tn += dij * phi[(size_t)j * np + p];
          if (kinetic) {                               /* h_KS phi_j of Eq. 16 with the kinetic operator: -1/2 lap phi_j */
            double lap = (hes[((size_t)0 * nnz + j) * np + p] + hes[((size_t)1 * nnz + j) * np + p]) + hes[((size_t)2 * nnz + j) * np + p];
            tk += dij * (-0.5 * lap);
          }
          if (g) {
            double Gj = 0.0;
            for (int c = 0; c < 3; c++) Gj += gp[c] * dphi[((size_t)c * nnz + j) * np + p];
            tg += dij * Gj;
          }
          if (Qb) tq += Qb[(size_t)i * nnz + j] * phi[(size_t)j * np + p];
        }
        double wp = S->w[p0 + p];
        double x = v[p0 + p] * tn + tg - tq + tk;
        static const int hx[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};   /* index of (c,e) in (xx,yy,zz,xy,xz,yz) */
        for (int c = 0; c < 3; c++) {
          double t = dphi[((size_t)c * nnz + i) * np + p] * x;
          if (g) {
            double hg = 0.0;
            for (int e = 0; e < 3; e++) hg += hes[((size_t)hx[c][e] * nnz + i) * np + p] * gp[e];
            t += hg * tn;
          }
          f[c] += 2.0 * wp * t;
        }
      }
      for (int c = 0; c < 3; c++) Frow[(size_t)i * 3 + c] = f[c];
    }
    for (int i = 0; i < nnz; i++)
      for (int c = 0; c < 3; c++) F[(size_t)fa[i] * 3 + c] += Frow[(size_t)i * 3 + c];
    free(Frow);
    free(Qb);
    free(Db);
    free(phi);
  }
  free(idx);
  free(afp);
}

/* brute-force Pulay forces (tiny inputs only): no batches, no culling, dense Dd, Qd [n_basis][n_basis] (Qd may be NULL),
 * written from Eq. 16 and Eq. 18 term by term with nabla_at phi_i = -grad phi_i:
 *   F_at = -2 sum_ij int [nabla_at phi_i] n_ij v phi_j + 2 sum_ij int [nabla_at phi_i] q_ij phi_j
 *          -2 sum_ij int [nabla_at phi_i] n_ij (g.grad phi_j) - 2 sum_ij int phi_i n_ij (g.nabla_at grad phi_j). */
void orc_brute_forces(const orc_system *S, const double *v, const double *g, const double *Dd, const double *Qd, int kinetic,
                      double *F) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nb = (int)afp[S->n_atoms];
  double *phi = (double *)malloc(sizeof(double) * (size_t)nb * 10);
  double *dph = phi + nb, *hes = phi + 4 * (size_t)nb;        /* dph[c*nb+i], hes[k*nb+i] */
  int *at_of = (int *)malloc(sizeof(int) * (size_t)nb);
  static const int hx[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};
  for (int64_t p = 0; p < S->n_points; p++) {
    int i = 0;
    for (int a = 0; a < S->n_atoms; a++) {
      int sp = S->atom_species[a];
      for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
        int l = S->shell_l[s];
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, a, s, S->xyz + 3 * p, val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++, i++) {
          phi[i] = val[m]; at_of[i] = a;
          for (int c = 0; c < 3; c++) dph[c * nb + i] = gr[m][c];
          for (int k = 0; k < 6; k++) hes[k * nb + i] = hh[m][k];
        }
      }
    }
    double wp = S->w[p];
    for (int a = 0; a < nb; a++)
      for (int b = 0; b < nb; b++) {
        double nab = Dd[(size_t)a * nb + b], qab = Qd ? Qd[(size_t)a * nb + b] : 0.0;
        double Gb = 0.0;
        if (g) for (int c = 0; c < 3; c++) Gb += g[(size_t)c * S->n_points + p] * dph[c * nb + b];
        for (int c = 0; c < 3; c++) {
          double nat_phi_a = -dph[c * nb + a];                       /* [nabla_at phi_a]_c for at = atom of a */
          F[at_of[a] * 3 + c] += wp * (-2.0 * nat_phi_a * nab * v[p] * phi[b] + 2.0 * nat_phi_a * qab * phi[b]);
          if (kinetic) F[at_of[a] * 3 + c] += wp * (-2.0 * nat_phi_a * nab * (-0.5 * ((hes[0 * nb + b] + hes[1 * nb + b]) + hes[2 * nb + b])));
          if (g) {
            F[at_of[a] * 3 + c] += wp * (-2.0 * nat_phi_a * nab * Gb);
            double nat_gb = 0.0;                                     /* g . nabla_at grad phi_b, component c, at = atom of b */
            for (int e = 0; e < 3; e++) nat_gb += -hes[hx[c][e] * nb + b] * g[(size_t)e * S->n_points + p];
            F[at_of[b] * 3 + c] += wp * (-2.0 * phi[a] * nab * nat_gb);
          }
        }
      }
  }
  free(at_of);
  free(phi);
  free(afp);
}

/* ====================================================================================================================
 * Kinetic term of h_KS (Eq. 4 L73 h_ij = <phi_i|h_KS|phi_j>, Eq. 24-27
 * L228-260, Fig. 6a "h_times_phi" then DSYR2K).  With (h phi_j)(r) = -1/2 lap phi_j(r) + v(r) phi_j(r) the batch
 * product K.L of Eq. 27 is not symmetric on the grid; Fig. 6a symmetrises it with DSYR2K, read here with alpha = 1/2
 * (reading P1b):
 *   h_ij[B] = 1/2 sum_{r in B} w(r) [ phi_i (h phi_j) + (h phi_i) phi_j ](r)   [+ the GGA term of O3, already symmetric].
 * lap phi is the trace of the Hessian of orc_shell_hess_at_point (pinned by finite differences in
 * tests/test_oracle_force_pins.py); the brute-force version below uses the radial form
 *   lap (R(d) Y_lm) = (R'' + 2 R'/d - l(l+1) R/d^2) Y_lm   instead, so that the two pin each other.
 * Further pins (tests/test_oracle_kinetic_pins.py): closed-form kinetic integrals of Gaussians; T symmetric positive
 * semidefinite; reduces to O3 for kinetic == 0.
 * ==================================================================================================================== */
void orc_integrate_hamiltonian_ks(const orc_system *S, int n_sel, const int32_t *batches, const double *v, const double *g,
                                  int kinetic, double *H_values) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (nnz == 0 || np == 0) continue;
    size_t sz = (size_t)nnz * np;
    double *phi = (double *)malloc(sizeof(double) * sz * 3);   /* phi, L = h phi, G = g . grad phi */
    double *Lp = phi + sz, *G = phi + 2 * sz;
    for (int i = 0; i < nnz;) {
      int l = S->shell_l[fs[i]];
      for (int p = 0; p < np; p++) {
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, fa[i], fs[i], S->xyz + 3 * (p0 + p), val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++) {
          size_t o = (size_t)(i + m) * np + p;
          double lap = (hh[m][0] + hh[m][1]) + hh[m][2];
          phi[o] = val[m];
          Lp[o] = v[p0 + p] * val[m];
          if (kinetic) Lp[o] += -0.5 * lap;
          double s = 0.0;
          if (g) for (int c = 0; c < 3; c++) s += g[(size_t)c * S->n_points + p0 + p] * gr[m][c];
          G[o] = s;
        }
      }
      i += 2 * l + 1;
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nnz; i++) {
      int A = fa[i];
      int ai = (int)(idx[i] - afp[A]);
      for (int j = 0; j < nnz; j++) {
        int B = fa[j];
        if (B < A) continue;
        int ld;
        int64_t off = find_block(S, A, B, &ld);
        if (off < 0) continue;
        int bj = (int)(idx[j] - afp[B]);
        double h = 0.0;
        for (int p = 0; p < np; p++) {
          double wp = S->w[p0 + p];
          double pi_ = phi[(size_t)i * np + p], pj = phi[(size_t)j * np + p];
          double term = 0.5 * wp * (pi_ * Lp[(size_t)j * np + p] + Lp[(size_t)i * np + p] * pj);
          if (g) term += wp * (G[(size_t)i * np + p] * pj + pi_ * G[(size_t)j * np + p]);
          h += term;
        }
        H_values[off + (int64_t)ai * ld + bj] += h;
      }
    }
    free(phi);
  }
  free(idx);
  free(afp);
}

/* brute force (tiny inputs only): dense Hd[n_basis][n_basis] = 1/2 sum_p w [phi_i (h phi_j) + (h phi_i) phi_j],
 * h phi = -1/2 (R'' + 2 R'/d - l(l+1) R/d^2) Y_lm + v phi, all functions x all points, no batches, no culling. */
void orc_brute_kinetic(const orc_system *S, const double *v, double *Hd) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nb = (int)afp[S->n_atoms];
  double *phi = (double *)malloc(sizeof(double) * (size_t)nb * 2);
  double *Lp = phi + nb;
  for (int64_t p = 0; p < S->n_points; p++) {
    int i = 0;
    for (int a = 0; a < S->n_atoms; a++) {
      int sp = S->atom_species[a];
      for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
        int l = S->shell_l[s];
        double rc = S->shell_rcut[s], dv[3];
        double d2 = dist2(S->xyz + 3 * p, S->atom_xyz + 3 * a, dv);
        double Y[7];
        double R = 0.0, dR = 0.0, d2R = 0.0, dd = 1.0;
        int inside = d2 < rc * rc;
        if (inside) {
          double d = sqrt(d2);
          double u[3] = {0.0, 0.0, 1.0};
          if (d > 0.0) { u[0] = dv[0] / d; u[1] = dv[1] / d; u[2] = dv[2] / d; }
          dd = d > S->r0 ? d : S->r0;
          orc_radial2(S, S->shell_spline[s], d, &R, &dR, &d2R);
          orc_solid_harmonics(l, u, Y, NULL);
        }
        for (int m = 0; m < 2 * l + 1; m++, i++) {
          phi[i] = inside ? R * Y[m] : 0.0;
          Lp[i] = inside ? -0.5 * (d2R + 2.0 * dR / dd - (double)(l * (l + 1)) * R / (dd * dd)) * Y[m] + v[p] * phi[i] : 0.0;
        }
      }
    }
    double wp = S->w[p];
    for (int a = 0; a < nb; a++)
      for (int c = 0; c < nb; c++) Hd[(size_t)a * nb + c] += 0.5 * wp * (phi[a] * Lp[c] + Lp[a] * phi[c]);
  }
  free(phi);
  free(afp);
}

/* ====================================================================================================================
 * Hessian of the density ("the Hessian matrix of the density,
 * d_xi d_xj n(r) (i, j = 1,...,3), is needed at least for total energy gradient calculations (forces and stresses) ...
 * straightforward extensions of Eq. (3) ... six components, and each component has the same cost as n(r) itself").
 * Differentiating Eq. 3 twice, for symmetric n_ij restricted to nnz(B):
 *   d_c d_e n(r) = 2 sum_ij n_ij [ (d_c d_e phi_i) phi_j + (d_c phi_i)(d_e phi_j) ](r),
 * components in the order (xx, yy, zz, xy, xz, yz).  Written as the double sum, no intermediate products.
 * Pins (tests/test_oracle_hessian_pins.py): central differences of the pinned grad n on displaced points; closed form for one
 * Gaussian; brute force over all functions in numpy; trace = Laplacian of n from the same pieces.
 * ==================================================================================================================== */
void orc_density_hessian(const orc_system *S, int n_sel, const int32_t *batches, const double *D_values, double *hess_n) {
  static const int ic[6] = {0, 1, 2, 0, 0, 1}, ie[6] = {0, 1, 2, 1, 2, 2};
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (np == 0) continue;
    size_t sz = (size_t)nnz * np;
    double *phi = (double *)malloc(sizeof(double) * (sz * 10 + 1));     /* phi, dphi[3], hess[6] */
    double *dphi = phi + sz, *hes = phi + 4 * sz;
    for (int i = 0; i < nnz;) {
      int l = S->shell_l[fs[i]];
      for (int p = 0; p < np; p++) {
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, fa[i], fs[i], S->xyz + 3 * (p0 + p), val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++) {
          phi[(size_t)(i + m) * np + p] = val[m];
          for (int c = 0; c < 3; c++) dphi[((size_t)c * nnz + i + m) * np + p] = gr[m][c];
          for (int k = 0; k < 6; k++) hes[((size_t)k * nnz + i + m) * np + p] = hh[m][k];
        }
      }
      i += 2 * l + 1;
    }
    double *Db = (double *)malloc(sizeof(double) * ((size_t)nnz * nnz + 1));
    restrict_matrix(S, afp, nnz, idx, fa, D_values, Db);
#pragma omp parallel for schedule(static)
    for (int p = 0; p < np; p++) {
      for (int k = 0; k < 6; k++) {
        int c = ic[k], e = ie[k];
        double acc = 0.0;
        for (int i = 0; i < nnz; i++)
          for (int j = 0; j < nnz; j++)
            acc += Db[(size_t)i * nnz + j] * (hes[((size_t)k * nnz + i) * np + p] * phi[(size_t)j * np + p] +
                                              dphi[((size_t)c * nnz + i) * np + p] * dphi[((size_t)e * nnz + j) * np + p]);
        hess_n[(size_t)k * S->n_points + p0 + p] = 2.0 * acc;
      }
    }
    free(Db);
    free(phi);
  }
  free(idx);
  free(afp);
}

/* ====================================================================================================================
 * Periodic boundary conditions: Bloch sums (Eq. 6-8, Eq. 11-12,
 * L113-115).  The real-space matrix h^uc_IJ (Eq. 12) runs over the N_rs functions -- the cell's functions and their
 * periodic images that are non-zero inside the cell at T = 0 -- and is integrated by O3 unchanged ("the exact same
 * real-space integration code", the points having been mapped back into the cell by the input generator).  Inserting
 * Eq. 7, chi_ik = sum_T e^{ik.T} phi_i(r - T), into Eq. 11 gives
 *   h_ij(k) = sum_{I image of i} sum_{J image of j} e^{ik.(T_J - T_I)} h^uc_IJ        (L115, "Bloch phase factors"),
 * and s_ij(k) analogously.  atom_home[A] < n_home is the cell atom that atom A is an image of (the cell's own atoms are
 * atoms 0..n_home-1 with T = 0), atom_T[A] its lattice translation.  Output: dense [n_hb][n_hb] real and imaginary parts,
 * n_hb = functions of the cell atoms.  Accumulated into (caller zeroes).
 * Pins (tests/test_oracle_periodic_pins.py): closed-form lattice sums of Gaussian overlaps; direct quadrature of Eq. 8 with
 * explicitly built Bloch functions; Hermitian, real at k = 0, positive definite; sum of weights = cell volume.
 * ==================================================================================================================== */
void orc_bloch_fold(const orc_system *S, const double *H_values, const int32_t *atom_home, const double *atom_T, int n_home,
                    const double *kpt, double *out_re, double *out_im) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int64_t nhb = afp[n_home];
  for (int A = 0; A < S->n_atoms; A++) {
    int nA = (int)(afp[A + 1] - afp[A]);
    for (int64_t q = S->row_ptr[A]; q < S->row_ptr[A + 1]; q++) {
      int B = S->col_atom[q];
      int nB = (int)(afp[B + 1] - afp[B]);
      int ld = S->blk_ld[q];
      double th = 0.0;
      for (int c = 0; c < 3; c++) th += kpt[c] * (atom_T[3 * B + c] - atom_T[3 * A + c]);
      double cs = cos(th), sn = sin(th);
      int64_t i0 = afp[atom_home[A]], j0 = afp[atom_home[B]];
      for (int a = 0; a < nA; a++)
        for (int b = 0; b < nB; b++) {
          double h = H_values[S->blk_off[q] + (int64_t)a * ld + b];
          out_re[(i0 + a) * nhb + (j0 + b)] += h * cs;
          out_im[(i0 + a) * nhb + (j0 + b)] += h * sn;
          if (A != B) {                         /* the stored block also stands for h^uc_JI = h^uc_IJ, phase conjugated */
            out_re[(j0 + b) * nhb + (i0 + a)] += h * cs;
            out_im[(j0 + b) * nhb + (i0 + a)] -= h * sn;
          }
        }
    }
  }
  free(afp);
}

/* ====================================================================================================================
 * tau matrix of meta-GGA functionals ("The evaluation of the tau matrix for
 * meta-GGAs has been omitted in (a) for brevity.  It is calculated via a single DGEMM ... and added to the h^uc_ij matrix
 * at the end of each batch").  The paper gives no formula; reading P1c takes the standard one: with the kinetic
 * energy density tau(r) = 1/2 sum_ij n_ij grad phi_i . grad phi_j and xi(r) = d f_xc / d tau supplied as a field,
 *   h_ij[B] += 1/2 sum_{r in B} w(r) xi(r) grad phi_i(r) . grad phi_j(r)          (= d/d n_ij of sum_r w f_xc(tau(r))).
 * Added into H_values (upper atom-pair blocks, diagonal blocks full), like O3.
 * Pins (tests/test_oracle_kinetic_pins.py): xi = 1 gives the kinetic matrix of the Laplacian form to grid accuracy
 * (integration by parts) and the numpy grad-grad matrix exactly; Tr(n M) = sum_r w xi tau; symmetric, PSD for xi > 0.
 * ==================================================================================================================== */
void orc_tau_matrix(const orc_system *S, int n_sel, const int32_t *batches, const double *xi, double *H_values) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (nnz == 0 || np == 0) continue;
    double *phi = (double *)malloc(sizeof(double) * (size_t)nnz * np * 4);
    double *dphi = phi + (size_t)nnz * np;
    orc_eval_basis(S, b, 1, nnz, fa, fs, fm, phi, dphi);
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nnz; i++) {
      int A = fa[i];
      int ai = (int)(idx[i] - afp[A]);
      for (int j = 0; j < nnz; j++) {
        int B = fa[j];
        if (B < A) continue;
        int ld;
        int64_t off = find_block(S, A, B, &ld);
        if (off < 0) continue;
        int bj = (int)(idx[j] - afp[B]);
        double h = 0.0;
        for (int p = 0; p < np; p++) {
          double gg = 0.0;
          for (int c = 0; c < 3; c++) gg += dphi[((size_t)c * nnz + i) * np + p] * dphi[((size_t)c * nnz + j) * np + p];
          h += 0.5 * S->w[p0 + p] * xi[p0 + p] * gg;
        }
        H_values[off + (int64_t)ai * ld + bj] += h;
      }
    }
    free(phi);
  }
  free(idx);
  free(afp);
}

/* ====================================================================================================================
 * Partition of unity (Eq. 21-22: the integration weight w(r) of a grid point
 * contains the atom-centred partition function, "a modified version of the partition function proposed by Stratmann et al."
 * cited at L190/L200 but not written out; reading P5 takes the textbook Stratmann-Scuseria-Frisch cell function):
 *   mu_AB = (d_A - d_B) / R_AB,  x = clamp(mu / 0.64, -1, 1),  z = (35 x - 35 x^3 + 21 x^5 - 5 x^7) / 16,  s = (1 - z) / 2,
 *   P_A(r) = prod_{B in cand(r), B != A} s(mu_AB),   w_A(r) = P_A(r) / sum_{B in cand(r)} P_B(r),
 * cand(r) = atoms within r_part of r (the O(N) neighbour restriction of L200).  out[p] = w_{owner[p]}(xyz[p]); 0 if the owner
 * is not a candidate.  Plain scans over all atoms, products in ascending atom order.
 * Pins (tests/test_oracle_partition_pins.py): sum over owners = 1 at arbitrary points; 1/2 on the bisecting plane of two atoms
 * and exactly 1 / 0 beyond mu = -+0.64; the polynomial's end values and symmetry s(mu) + s(-mu) = 1; rigid motions.
 * ==================================================================================================================== */
static double orc_stratmann_s(double mu) {
  double x = mu / 0.64;
  if (x <= -1.0) return 1.0;
  if (x >= 1.0) return 0.0;
  double z = (35.0 * x - 35.0 * x * x * x + 21.0 * x * x * x * x * x - 5.0 * x * x * x * x * x * x * x) / 16.0;
  double s = 0.5 * (1.0 - z);
  if (s < 0.0) s = 0.0;
  if (s > 1.0) s = 1.0;
  return s;
}

void orc_partition_weights(const orc_system *S, int64_t n, const double *xyz, const int32_t *owner, double r_part, double *out) {
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t p = 0; p < n; p++) {
    const double *r = xyz + 3 * p;
    double sum = 0.0, pown = 0.0;
    for (int A = 0; A < S->n_atoms; A++) {
      const double *Ra = S->atom_xyz + 3 * A;
      double dA = sqrt((r[0] - Ra[0]) * (r[0] - Ra[0]) + (r[1] - Ra[1]) * (r[1] - Ra[1]) + (r[2] - Ra[2]) * (r[2] - Ra[2]));
      if (dA > r_part) continue;
      double P = 1.0;
      for (int B = 0; B < S->n_atoms; B++) {
        if (B == A) continue;
        const double *Rb = S->atom_xyz + 3 * B;
        double dB = sqrt((r[0] - Rb[0]) * (r[0] - Rb[0]) + (r[1] - Rb[1]) * (r[1] - Rb[1]) + (r[2] - Rb[2]) * (r[2] - Rb[2]));
        if (dB > r_part) continue;
        double Rab = sqrt((Ra[0] - Rb[0]) * (Ra[0] - Rb[0]) + (Ra[1] - Rb[1]) * (Ra[1] - Rb[1]) + (Ra[2] - Rb[2]) * (Ra[2] - Rb[2]));
        P *= orc_stratmann_s((dA - dB) / Rab);
      }
      sum += P;
      if (A == owner[p]) pown = P;
    }
    out[p] = sum > 0.0 ? pown / sum : 0.0;
  }
}

/* ====================================================================================================================
 * O9  Pulay part of the stress tensor (Eq. 20: sigma_lm = (1/V) dE_tot/d eps_lm;
 * L299-308: force AND stress components are the same per-batch dense products; L405: the Pulay contribution to F_at and
 * sigma_lm is evaluated alongside the density update; L413-415 / Table 2: "SCF+F+sigma" is the paper's largest case).
 * The paper defers the individual terms to its Ref. [83] (L158); what it does fix is the handle, Eq. 20, and that is what is
 * written out here -- exactly as the forces above follow from Eq. 14 (reading P22).  Under a homogeneous strain
 * r -> (1 + eps) r of atoms AND grid points, a basis function seen from a grid point becomes phi_i((1 + eps)(r - R_at)), so
 *   d phi_i / d eps_lm = (d_l phi_i) (r - R_at)_m ,     d (d_c phi_i) / d eps_lm = (d_l d_c phi_i) (r - R_at)_m ,
 * and the Pulay part of Eq. 20 is the derivative of  Tr(n h(eps)) - Tr(q s(eps))  at fixed n_ij, q_ij (Eq. 17) and fixed
 * point values v_p, g_p, w_p (the strain dependence of the integration weights and of the fields belongs to the other terms
 * of the stress, which like the Hellmann-Feynman and multipole forces are not on this path):
 *   V sigma_lm = 2 sum_p w_p sum_i (r_p - R_at(i))_m { d_l phi_i [ sum_j n_ij (v_p phi_j + g_p.grad phi_j [- 1/2 lap phi_j]) - q_ij phi_j ]
 *                                                      + (Hess phi_i g_p)_l sum_j n_ij phi_j } ,
 * i.e. the force integrand of O5 weighted with the distance vector to the function's own atom.  With point-attached fields
 * that do not co-rotate, sigma need not be symmetric; all nine components are returned, sigma[l][m].
 * Pins (tests/test_oracle_stress_pins.py): central differences of the already pinned H and S on a strained copy of the
 * inputs; the term-by-term brute force below (no batches, no culling, both index orders written out); sum rule with the
 * forces for an s-only basis; invariance under translation of the whole system and under re-batching; linear in (n, q).
 * kinetic != 0 (the -1/2 lap phi_j inside h_KS phi_j, as in O5/Eq. 16) is the PULAY part of the kinetic stress: the derivative
 * of the basis-function factors only.  Its pins: orc_brute_stress_ks (radial-form Laplacian, both index orders), additivity
 * sigma(v, kin) = sigma(v, off) + sigma(0, kin), and central differences of Tr(n t(eps)) of the pinned kinetic matrix, which
 * equal sigma(0, kin) + sum_ij n_ij <phi_i| d_l d_m |phi_j> to grid accuracy (the commutator [t, x_m d_l] = -d_l d_m; that
 * second term is the kinetic stress proper and, like the Hellmann-Feynman terms, not on this path).
 * ==================================================================================================================== */
void orc_pulay_stress(const orc_system *S, int n_sel, const int32_t *batches, const double *v, const double *g,
                      const double *D_values, const double *Q_values, int kinetic, double volume, double *sigma) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nf_tot = (int)afp[S->n_atoms];
  int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)nf_tot);
  int32_t *fa = idx + nf_tot, *fs = fa + nf_tot, *fm = fs + nf_tot;
  static const int hx[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};   /* index of (c,e) in (xx,yy,zz,xy,xz,yz) */
  for (int q = 0; q < n_sel; q++) {
    int b = batches[q];
    int64_t p0 = S->batch_ptr[b];
    int np = (int)(S->batch_ptr[b + 1] - p0);
    int nnz = orc_batch_nnz(S, b, idx, fa, fs, fm);
    if (nnz == 0 || np == 0) continue;
    size_t sz = (size_t)nnz * np;
    double *phi = (double *)malloc(sizeof(double) * sz * 10);     /* phi, dphi[3], hess[6] */
    double *dphi = phi + sz, *hes = phi + 4 * sz;
    for (int i = 0; i < nnz;) {
      int l = S->shell_l[fs[i]];
      for (int p = 0; p < np; p++) {
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, fa[i], fs[i], S->xyz + 3 * (p0 + p), val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++) {
          phi[(size_t)(i + m) * np + p] = val[m];
          for (int c = 0; c < 3; c++) dphi[((size_t)c * nnz + i + m) * np + p] = gr[m][c];
          for (int k = 0; k < 6; k++) hes[((size_t)k * nnz + i + m) * np + p] = hh[m][k];
        }
      }
      i += 2 * l + 1;
    }
    double *Db = (double *)malloc(sizeof(double) * (size_t)nnz * nnz);
    double *Qb = Q_values ? (double *)malloc(sizeof(double) * (size_t)nnz * nnz) : NULL;
    restrict_matrix(S, afp, nnz, idx, fa, D_values, Db);
    if (Qb) restrict_matrix(S, afp, nnz, idx, fa, Q_values, Qb);
    double *Srow = (double *)calloc((size_t)nnz * 9, sizeof(double));     /* per-function contribution, summed below */
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nnz; i++) {
      double s9[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
      const double *Ra = S->atom_xyz + 3 * fa[i];
      for (int p = 0; p < np; p++) {
        double gp[3] = {0.0, 0.0, 0.0};
        if (g) for (int c = 0; c < 3; c++) gp[c] = g[(size_t)c * S->n_points + p0 + p];
        double tn = 0.0, tg = 0.0, tq = 0.0, tk = 0.0;
        for (int j = 0; j < nnz; j++) {
          double dij = Db[(size_t)i * nnz + j];
          tn += dij * phi[(size_t)j * np + p];
          if (kinetic) {
            double lap = (hes[((size_t)0 * nnz + j) * np + p] + hes[((size_t)1 * nnz + j) * np + p]) + hes[((size_t)2 * nnz + j) * np + p];
            tk += dij * (-0.5 * lap);
          }
          if (g) {
            double Gj = 0.0;
            for (int c = 0; c < 3; c++) Gj += gp[c] * dphi[((size_t)c * nnz + j) * np + p];
            tg += dij * Gj;
          }
          if (Qb) tq += Qb[(size_t)i * nnz + j] * phi[(size_t)j * np + p];
        }
        double wp = S->w[p0 + p];
        double x = v[p0 + p] * tn + tg - tq + tk;
        for (int l = 0; l < 3; l++) {
          double t = dphi[((size_t)l * nnz + i) * np + p] * x;
          if (g) {
            double hg = 0.0;
            for (int e = 0; e < 3; e++) hg += hes[((size_t)hx[l][e] * nnz + i) * np + p] * gp[e];
            t += hg * tn;
          }
          for (int m = 0; m < 3; m++) s9[l][m] += 2.0 * wp * t * (S->xyz[3 * (p0 + p) + m] - Ra[m]);
        }
      }
      for (int l = 0; l < 3; l++)
        for (int m = 0; m < 3; m++) Srow[(size_t)i * 9 + 3 * l + m] = s9[l][m];
    }
    for (int i = 0; i < nnz; i++)
      for (int k = 0; k < 9; k++) sigma[k] += Srow[(size_t)i * 9 + k] / volume;
    free(Srow);
    free(Qb);
    free(Db);
    free(phi);
  }
  free(idx);
  free(afp);
}

/* brute-force Pulay stress (tiny inputs only): no batches, no culling, dense Dd, Qd (Qd may be NULL).  d/d eps_lm of
 *   sum_ab n_ab int [ phi_a v phi_b + g.(grad phi_a phi_b + phi_a grad phi_b) (+ 1/2 (phi_a t phi_b + t phi_a phi_b)) ] - sum_ab q_ab int phi_a phi_b
 * with every strained factor differentiated separately (both index orders written out, nothing symmetrised by hand). */
void orc_brute_stress(const orc_system *S, const double *v, const double *g, const double *Dd, const double *Qd, double volume,
                      double *sigma) {
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nb = (int)afp[S->n_atoms];
  double *phi = (double *)malloc(sizeof(double) * (size_t)nb * 10);
  double *dph = phi + nb, *hes = phi + 4 * (size_t)nb;        /* dph[c*nb+i], hes[k*nb+i] */
  int *at_of = (int *)malloc(sizeof(int) * (size_t)nb);
  static const int hx[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};
  for (int64_t p = 0; p < S->n_points; p++) {
    int i = 0;
    for (int a = 0; a < S->n_atoms; a++) {
      int sp = S->atom_species[a];
      for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
        int l = S->shell_l[s];
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, a, s, S->xyz + 3 * p, val, gr, hh);
        for (int m = 0; m < 2 * l + 1; m++, i++) {
          phi[i] = val[m]; at_of[i] = a;
          for (int c = 0; c < 3; c++) dph[c * nb + i] = gr[m][c];
          for (int k = 0; k < 6; k++) hes[k * nb + i] = hh[m][k];
        }
      }
    }
    double wp = S->w[p];
    for (int a = 0; a < nb; a++)
      for (int b = 0; b < nb; b++) {
        double nab = Dd[(size_t)a * nb + b], qab = Qd ? Qd[(size_t)a * nb + b] : 0.0;
        if (nab == 0.0 && qab == 0.0) continue;
        const double *Ra = S->atom_xyz + 3 * at_of[a], *Rb = S->atom_xyz + 3 * at_of[b];
        for (int l = 0; l < 3; l++)
          for (int m = 0; m < 3; m++) {
            double da = S->xyz[3 * p + m] - Ra[m], db = S->xyz[3 * p + m] - Rb[m];
            double dphi_a = dph[l * nb + a] * da, dphi_b = dph[l * nb + b] * db;     /* d phi / d eps_lm */
            double t = (nab * v[p] - qab) * (dphi_a * phi[b] + phi[a] * dphi_b);
            if (g) {
              double Ga = 0.0, Gb = 0.0, dGa = 0.0, dGb = 0.0;                        /* g.grad phi and its strain derivative */
              for (int c = 0; c < 3; c++) {
                double gc = g[(size_t)c * S->n_points + p];
                Ga += gc * dph[c * nb + a]; Gb += gc * dph[c * nb + b];
                dGa += gc * hes[hx[l][c] * nb + a] * da; dGb += gc * hes[hx[l][c] * nb + b] * db;
              }
              t += nab * (dGa * phi[b] + Ga * dphi_b + dphi_a * Gb + phi[a] * dGb);
            }
            sigma[3 * l + m] += wp * t / volume;
          }
      }
  }
  free(at_of);
  free(phi);
  free(afp);
}

/* brute-force Pulay stress WITH the kinetic operator (tiny inputs only): orc_brute_stress plus the kinetic part of
 * orc_pulay_stress written independently -- no batches, no culling, both index orders of the symmetrised product
 * 1/2 (phi_a t phi_b + t phi_a phi_b) written out, and t phi taken in the RADIAL form
 *   t (R(d) Y_lm) = -1/2 (R'' + 2 R'/d - l(l+1) R/d^2) Y_lm        (as orc_brute_kinetic does)
 * instead of the trace of the Cartesian Hessian that orc_pulay_stress uses, so that the two pin each other.
 * What is differentiated is the PULAY part ("the Pulay contribution to F_at and sigma_lm"): the strain derivative
 * of the basis-function factor, d phi_a / d eps_lm = (d_l phi_a)(r - R_a)_m, with t phi_b held as the force expression of Eq. 16
 * holds h_KS phi_j:
 *   V sigma^kin_lm = sum_p w_p sum_ab n_ab [ (d phi_a / d eps_lm) (t phi_b) + (t phi_a) (d phi_b / d eps_lm) ] .
 * The derivative of the operator's own factor, x_m d_l (t phi_b), is not a Pulay term; by [t, x_m d_l] = -d_l d_m it differs
 * from the above by  sum_ab n_ab <phi_a| d_l d_m |phi_b>  (the kinetic stress proper), which tests/test_oracle_stress_pins.py
 * adds when it compares with finite differences of Tr(n t(eps)). */
void orc_brute_stress_ks(const orc_system *S, const double *v, const double *g, const double *Dd, const double *Qd, int kinetic,
                         double volume, double *sigma) {
  orc_brute_stress(S, v, g, Dd, Qd, volume, sigma);
  if (!kinetic) return;
  int64_t *afp = (int64_t *)malloc(sizeof(int64_t) * (S->n_atoms + 1));
  orc_atom_fn_ptr(S, afp);
  int nb = (int)afp[S->n_atoms];
  double *phi = (double *)malloc(sizeof(double) * (size_t)nb * 5);
  double *dph = phi + nb, *tph = phi + 4 * (size_t)nb;        /* dph[c*nb+i], tph[i] = (t phi_i)(r_p) */
  int *at_of = (int *)malloc(sizeof(int) * (size_t)nb);
  for (int64_t p = 0; p < S->n_points; p++) {
    int i = 0;
    for (int a = 0; a < S->n_atoms; a++) {
      int sp = S->atom_species[a];
      for (int s = S->species_shell_ptr[sp]; s < S->species_shell_ptr[sp + 1]; s++) {
        int l = S->shell_l[s];
        double val[7], gr[7][3], hh[7][6];
        orc_shell_hess_at_point(S, a, s, S->xyz + 3 * p, val, gr, hh);     /* phi and grad phi (pinned by finite differences) */
        double rc = S->shell_rcut[s], dv[3];
        double d2 = dist2(S->xyz + 3 * p, S->atom_xyz + 3 * a, dv);
        double Y[7];
        double R = 0.0, dR = 0.0, d2R = 0.0, dd = 1.0;
        int inside = d2 < rc * rc;
        if (inside) {
          double d = sqrt(d2);
          double u[3] = {0.0, 0.0, 1.0};
          if (d > 0.0) { u[0] = dv[0] / d; u[1] = dv[1] / d; u[2] = dv[2] / d; }
          dd = d > S->r0 ? d : S->r0;
          orc_radial2(S, S->shell_spline[s], d, &R, &dR, &d2R);
          orc_solid_harmonics(l, u, Y, NULL);
        }
        for (int m = 0; m < 2 * l + 1; m++, i++) {
          phi[i] = val[m]; at_of[i] = a;
          for (int c = 0; c < 3; c++) dph[c * nb + i] = gr[m][c];
          tph[i] = inside ? -0.5 * (d2R + 2.0 * dR / dd - (double)(l * (l + 1)) * R / (dd * dd)) * Y[m] : 0.0;
        }
      }
    }
    double wp = S->w[p];
    for (int a = 0; a < nb; a++)
      for (int b = 0; b < nb; b++) {
        double nab = Dd[(size_t)a * nb + b];
        if (nab == 0.0) continue;
        const double *Ra = S->atom_xyz + 3 * at_of[a], *Rb = S->atom_xyz + 3 * at_of[b];
        for (int l = 0; l < 3; l++)
          for (int m = 0; m < 3; m++) {
            double dphi_a = dph[l * nb + a] * (S->xyz[3 * p + m] - Ra[m]);     /* d phi_a / d eps_lm */
            double dphi_b = dph[l * nb + b] * (S->xyz[3 * p + m] - Rb[m]);
            sigma[3 * l + m] += wp * nab * (dphi_a * tph[b] + tph[a] * dphi_b) / volume;
          }
      }
  }
  free(at_of);
  free(phi);
  free(afp);
}
