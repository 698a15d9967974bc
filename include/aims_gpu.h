/* aims_gpu.h -- C ABI of the B200-native real-space grid operations of arXiv:1912.06636
 * (Huhn, Lange, Yu, Yoon, Blum: "GPGPU acceleration of all-electron electronic structure theory using localized
 * numeric atom-centered basis functions").  Citations: PAPER.md L<line> = /root/reference/PAPER.md.
 *
 * The three hot calls follow the paper's statement of the problem (Fig. 6):
 *   aims_gpu_eval_basis             "calculate_phi" on the reduced subspace nnz(B) of every batch   (L235, L314, L322)
 *   aims_gpu_integrate_hamiltonian  h_ij = sum_B sum_{r in B} w(r) phi_i(r) (h phi_j)(r)             (Eq. 23-27)
 *   aims_gpu_update_density         n(r) = sum_ij phi_i(r) n_ij phi_j(r) and grad n                  (Eq. 3)
 * Every step runs in hand-written sm_100a kernels; there is no CPU fallback and no other backend.
 *
 * Conventions
 *  - All functions return AIMS_OK (0) or a negative aims_status; they never throw (every entry point catches C++
 *    exceptions of its host-side bookkeeping: std::bad_alloc -> AIMS_ERR_NOMEM), exit or print.
 *  - HOST pointers are read during the call that receives them and may be freed afterwards.
 *    DEVICE pointers must be valid on the context's device, 16-byte aligned, and are owned by the caller.
 *  - Work is enqueued on the stream given at creation.  Outputs are valid once the caller has synchronised that
 *    stream.  Errors detectable at enqueue time are returned; an asynchronous CUDA fault surfaces at the next
 *    call or at destroy (AIMS_ERR_CUDA, text in aims_gpu_last_error).  Device-side capacity / consistency flags raised
 *    by a hot call are reported ONLY by aims_gpu_synchronize (once; the flag is then cleared).
 *  - Global basis index: atom-major, then the species' shells in order, then m = -l..l.
 *  - Lengths are in Angstrom; nothing converts units.
 *  - One context per host thread; a context is not thread-safe.  Several contexts may be alive at once (also on one device).
 *
 * Deviations from the signatures sketched in SURVEY.md 8(b), and why:
 *  - aims_gpu_create takes `workspace_bytes`: Phi planes of the whole grid do not fit in HBM (config 5: 54 GB per plane), so
 *    every call streams them through a workspace in chunks of batches; its size is the caller's to bound.
 *  - aims_gpu_basis_sizes / aims_gpu_eval_basis have no `want_grad`: a NULL `dphi` is the flag, and the sizes do not depend
 *    on it (dphi is 3 * n_phi).
 * The diagnostic entry points (timing, launch count, FP64 probes) are grouped at the end of this header; nothing on the
 * product path needs them.
 */
#ifndef AIMS_GPU_H
#define AIMS_GPU_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  AIMS_OK = 0,
  AIMS_ERR_INVALID_ARG = -1, /* NULL where not allowed, inconsistent sizes, batch range outside [0, n_batches] */
  AIMS_ERR_CUDA = -2,        /* a CUDA runtime call failed; see aims_gpu_last_error */
  AIMS_ERR_NOMEM = -3,       /* device workspace could not be allocated */
  AIMS_ERR_UNSUPPORTED = -4  /* l > 3, > 32 shells per species, > AIMS_MAX_ACTIVE_ATOMS atoms touching one batch, ... */
} aims_status;

#define AIMS_MAX_L 3
#define AIMS_MAX_SHELLS_PER_SPECIES 32
#define AIMS_MAX_ACTIVE_ATOMS 96 /* atoms whose cutoff sphere reaches one batch */

/* Basis: numeric atom-centred functions phi = R_s(d) Y_lm(u) (readings P8-P11).
 * R_s is DEFINED by the spline table: t = ln(max(d,r0)/r0)/log_inc, k = min(floor t, n_knots-2), x = t-k,
 * R = a + x(b + x(c + x d)); phi is exactly 0 where |r-R_a|^2 >= rcut^2.  HOST pointers. */
typedef struct {
  int32_t n_atoms, n_species, n_shells, n_splines, n_knots;
  const double *atom_xyz;           /* [n_atoms][3] */
  const int32_t *atom_species;      /* [n_atoms], 0..n_species-1 */
  const int32_t *species_shell_ptr; /* [n_species+1]: shells species_shell_ptr[s] .. species_shell_ptr[s+1]-1 */
  const int32_t *shell_l;           /* [n_shells], 0..AIMS_MAX_L */
  const double *shell_rcut;         /* [n_shells] */
  const int32_t *shell_spline;      /* [n_shells], index into spline_coef */
  double r0, log_inc;               /* knots r_k = r0 exp(log_inc k), k = 0..n_knots-1 */
  const double *spline_coef;        /* [n_splines][n_knots-1][4] = (a,b,c,d) per interval */
} aims_basis_desc;

/* Integration grid cut into spatially compact batches.  The points of batch b are
 * xyz[batch_ptr[b] .. batch_ptr[b+1]); the library never re-batches.  HOST pointers. */
typedef struct {
  int64_t n_points;
  int32_t n_batches;
  int32_t max_batch_points;         /* >= every batch size */
  const double *xyz;                /* [n_points][3] */
  const double *w;                  /* [n_points] integration weight w(r) of Eq. 21 */
  const int64_t *batch_ptr;         /* [n_batches+1], ascending, batch_ptr[0] = 0 */
} aims_grid_desc;

/* Atom-pair block-sparse layout of H, S and D (replaces the paper's "locally-indexed dense" storage, L291-297;
 * SURVEY.md reading P13).  Only blocks with col_atom >= row atom are stored; block q of row A is row-major
 * [n_fn(A)][blk_ld[q]] at values[blk_off[q]]; diagonal blocks (A,A) hold the full square.  Pairs absent from
 * the pattern are treated as exactly zero.  blk_off and blk_ld must be even (16-byte rows).  HOST pointers. */
typedef struct {
  int32_t n_block_rows;             /* == n_atoms */
  const int64_t *row_ptr;           /* [n_atoms+1] */
  const int32_t *col_atom;          /* [n_blocks], ascending within a row */
  const int64_t *blk_off;           /* [n_blocks] */
  const int32_t *blk_ld;            /* [n_blocks], >= n_fn(col_atom) */
  int64_t n_values;
} aims_bsr_desc;

typedef struct aims_gpu_ctx aims_gpu_ctx;

/* Create a context on `device` (cudaSetDevice ordinal) that enqueues on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = legacy default stream).  Copies the three descriptions to the
 * device, runs the culling once to size every per-batch list, and allocates workspaces (at most
 * workspace_bytes for the per-chunk Phi planes, never less than one batch in every plane layout; 0 = default 24 GiB,
 * clamped to free memory).  Synchronises the stream before returning.
 * On failure *out is NULL (nothing to free) or a half-built context that accepts ONLY aims_gpu_last_error and
 * aims_gpu_destroy -- the caller must still destroy it. */
int aims_gpu_create(aims_gpu_ctx **out, const aims_basis_desc *basis, const aims_grid_desc *grid,
                    const aims_bsr_desc *bsr, int device, void *cuda_stream, int64_t workspace_bytes);
int aims_gpu_destroy(aims_gpu_ctx *ctx);
/* Text of the last error on this context (ctx-owned, valid until the next call); "" if none. ctx may be NULL. */
const char *aims_gpu_last_error(const aims_gpu_ctx *ctx);

/* Sizes of the outputs of aims_gpu_eval_basis for batches [b0,b1): n_index = sum nnz(B), n_phi = sum nnz(B)*|B|.
 * HOST outputs. */
int aims_gpu_basis_sizes(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, int64_t *n_index, int64_t *n_phi);

/* Step 1 (S1a+S1b).  For each batch b in [b0,b1): the ascending list of global indices of nnz(B_b) (
 * i in nnz(B) iff some point p of B has ((dx*dx+dy*dy)+dz*dz) < rcut*rcut, decided per shell in separately rounded
 * IEEE operations, reading P6), and phi (and grad phi if dphi != NULL) of those functions at the batch's points.
 * DEVICE outputs, caller-sized with aims_gpu_basis_sizes:
 *   fn_ptr  [b1-b0+1]  fn_index[fn_ptr[k] .. fn_ptr[k+1]) belongs to batch b0+k
 *   fn_index[n_index]
 *   phi_ptr [b1-b0+1]  phi[phi_ptr[k] + i*n_p + p], i < nnz, p < n_p = |B| (point index fastest)
 *   phi     [n_phi]
 *   dphi    NULL or [3*n_phi]: d phi/d x_c at dphi[3*phi_ptr[k] + (c*nnz + i)*n_p + p] */
int aims_gpu_eval_basis(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, int64_t *fn_ptr, int32_t *fn_index,
                        int64_t *phi_ptr, double *phi, double *dphi);

/* Step 2 (S2a-S2d).  H_values (+)= sum over batches [b0,b1) of
 *     sum_p w_p phi_i(r_p) v_p phi_j(r_p)  +  [g != NULL]  sum_p w_p g_p . (grad phi_i phi_j + phi_i grad phi_j)(r_p)
 * for i,j in nnz(B), scattered into the block pattern (Eq. 23-27; GGA term in the integrated-by-parts form, L67 and
 * Eq. 18, reading P2).  Overlap matrix: pass v = 1.  DEVICE pointers:
 *   v [n_points] (may be NULL only if n_points == 0), g NULL or [3][n_points] (component-major), H_values [n_values].
 * accumulate == 0: H_values is zeroed first; != 0: added to (Eq. 28-29 partial sums). */
int aims_gpu_integrate_hamiltonian(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *v, const double *g,
                                   double *H_values, int accumulate);

/* Row f2 of SURVEY.md 8(f): the full h_KS phi of Eq. 26 with the kinetic operator, "h_times_phi" of
 * Fig. 6a (L323).  kinetic != 0:  (h phi_j)(r) = -1/2 lap phi_j(r) + v(r) phi_j(r); the batch product K.L of Eq. 27 is then
 * not symmetric on the grid and is symmetrised as Fig. 6a does with DSYR2K (alpha = 1/2, reading P1b):
 *   H_values (+)= sum_p w_p { 1/2 [phi_i (h phi_j) + (h phi_i) phi_j] + [g != NULL] g_p . grad(phi_i phi_j) }(r_p).
 * lap (R(d) Y_lm) = (R'' + 2 R'/d - l(l+1) R/d^2) Y_lm with R'' from the same spline table.  kinetic == 0: identical to
 * aims_gpu_integrate_hamiltonian.  Arguments as there. */
int aims_gpu_integrate_hamiltonian_ks(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *v, const double *g,
                                      int kinetic, double *H_values, int accumulate);

/* Row f2, meta-GGA: the "tau matrix" of PAPER.md L377 ("calculated via a single DGEMM ... and added to the h^uc_ij matrix at
 * the end of each batch"; the paper gives no formula, reading P1c):
 *   H_values += sum over batches [b0,b1) of  1/2 sum_p w_p xi_p grad phi_i(r_p) . grad phi_j(r_p),   xi = d f_xc / d tau.
 * Always accumulates.  DEVICE pointers: xi [n_points], H_values [n_values]. */
int aims_gpu_add_tau_matrix(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *xi, double *H_values);

/* Step 3 (S3a-S3d).  For every point p of batches [b0,b1):  n[p] = sum_ij phi_i D_ij phi_j,
 * grad_n[c][p] = 2 sum_ij d_c phi_i D_ij phi_j (D symmetric), i,j in nnz(B) (Eq. 3; Fig. 6b).
 * DEVICE pointers: D_values [n_values] in the pattern of aims_bsr_desc (upper blocks; the symmetric full matrix is
 * implied), n [n_points], grad_n NULL or [3][n_points].  Points of other batches are not touched. */
int aims_gpu_update_density(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *D_values, double *n,
                            double *grad_n);

/* Row f1 of SURVEY.md 8(f): Hessian of the density, needed for total-energy gradients.  For every point
 * p of batches [b0,b1), with symmetric n_ij restricted to nnz(B):
 *   hess_n[k][p] = 2 sum_ij n_ij [ (d_c d_e phi_i) phi_j + (d_c phi_i)(d_e phi_j) ](r_p),  k = (c,e) in (xx, yy, zz, xy, xz, yz).
 * DEVICE pointers: D_values [n_values] (pattern of aims_bsr_desc), hess_n [6][n_points] (component-major).  Points of other
 * batches are not touched.  Reduced without atomics: bitwise reproducible.  Timed under slot [5] of aims_gpu_timing_read. */
int aims_gpu_density_hessian(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *D_values, double *hess_n);

/* Row f1 of SURVEY.md 8(f): Pulay forces, evaluated on the same batches as the density update (Eq. 14-18
 * L129-150; L301-308; L405).  For the reduced h_KS of this library (local potential v plus the GGA term above) and
 * nabla_at phi_i = -grad phi_i for the functions i centred on atom `at`, Eq. 16 and Eq. 18 on the grid:
 *   F[at][c] (+)= 2 sum_{p in batches [b0,b1)} w_p sum_{i on at} sum_j
 *        { d_c phi_i [ n_ij (v_p phi_j + g_p . grad phi_j) - q_ij phi_j ]  +  (Hess phi_i g_p)_c n_ij phi_j }   (at r_p)
 * = -d/dR_at [ Tr(n h(R)) - Tr(q s(R)) ] at fixed n_ij, q_ij, v, g, weights and grid.  The Hellmann-Feynman, multipole and
 * atomic-ZORA terms (L403, Eq. 19) are not on this path.  DEVICE pointers:
 *   v [n_points]; g NULL (no GGA term) or [3][n_points]; D_values [n_values] = n_ij and Q_values NULL or [n_values] =
 *   the energy-weighted density matrix q_ij of Eq. 17, both in the pattern of aims_bsr_desc (symmetric, upper blocks);
 *   F [n_atoms][3].  accumulate == 0: F is zeroed first.  F is accumulated with floating-point atomics: two runs agree
 *   to rounding, not bitwise. */
int aims_gpu_pulay_forces(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *v, const double *g,
                          const double *D_values, const double *Q_values, double *F, int accumulate);

/* aims_gpu_pulay_forces with the h_KS phi_j of Eq. 16 carrying the kinetic operator when kinetic != 0:
 * v_p phi_j -> v_p phi_j - 1/2 lap phi_j(r_p) in the formula above (rows f1 + f2).  Eq. 16 uses the Hermiticity of h_KS,
 * which the grid quadrature reproduces only to its own accuracy for -1/2 lap: that part is the gradient of Tr(n t(R)) to
 * grid accuracy.  kinetic == 0: identical to aims_gpu_pulay_forces. */
int aims_gpu_pulay_forces_ks(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                             const double *D_values, const double *Q_values, double *F, int accumulate);

/* Row f1 of SURVEY.md 8(f), stress: the Pulay contribution to the stress tensor, evaluated in the same pass as the Pulay
 * forces (Eq. 20: sigma_lm = (1/V) dE_tot/d eps_lm; L299-308; L405 "the Pulay contribution to F_at and
 * sigma_lm"; Table 2 "SCF+F+sigma").  The paper defers the terms to its Ref. [83]; reading P22 takes Eq. 20 itself:
 * under a homogeneous strain r -> (1 + eps) r of atoms and grid points, at fixed n_ij, q_ij and fixed point values v_p, g_p, w_p,
 *   sigma[l][m] (+)= (2 / volume) sum_{p in batches [b0,b1)} w_p sum_i (r_p - R_at(i))_m
 *        { d_l phi_i [ sum_j n_ij (h_KS phi_j) - q_ij phi_j ]  +  (Hess phi_i g_p)_l sum_j n_ij phi_j }   (at r_p),
 * = (1/volume) d/d eps_lm [ Tr(n h(eps)) - Tr(q s(eps)) ], i.e. the force integrand weighted with the distance vector to the
 * function's own atom; (h_KS phi_j) = v phi_j + g.grad phi_j (- 1/2 lap phi_j if kinetic != 0) as in aims_gpu_pulay_forces_ks.
 * For the kinetic part this is the PULAY term only (derivative of the basis-function factors); d/d eps_lm Tr(n t(eps)) has in
 * addition sum_ij n_ij <phi_i| d_l d_m |phi_j> from the operator itself, which the caller adds with the other non-Pulay terms.
 * Point-attached fields do not co-rotate, so sigma need not be symmetric: all nine components are returned.
 * volume: the cell volume V (> 0; pass 1 for a cluster to obtain dE/d eps).  DEVICE pointers as in aims_gpu_pulay_forces_ks,
 * plus sigma [3][3]; F may be NULL (stress only).  accumulate == 0: F and sigma are zeroed first.  Accumulated with
 * floating-point atomics (reruns agree to rounding). */
int aims_gpu_pulay_forces_stress(aims_gpu_ctx *ctx, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                                 const double *D_values, const double *Q_values, double volume, double *F, double *sigma,
                                 int accumulate);

/* Row f4 of SURVEY.md 8(f): the partition-of-unity factor of the integration weights w(r) (Eq. 21-22; the
 * paper cites "a modified version of the partition function proposed by Stratmann et al." without writing it out; DESIGN.md
 * reading P5 takes the textbook Stratmann-Scuseria-Frisch cell function with a = 0.64, restricted to the atoms within r_part
 * of the point):  w_part[p] = P_owner(r_p) / sum_{A in cand(r_p)} P_A(r_p),  P_A = prod_{B in cand, B != A} s(mu_AB),
 * mu_AB = (|r-R_A| - |r-R_B|) / |R_A-R_B|, cand(r) = atoms with sqrt((dx*dx + dy*dy) + dz*dz) <= r_part in separately rounded IEEE
 * operations (a discrete decision, as in reading P6); 0 if the owner is not a candidate.  The atoms are
 * the context's.  DEVICE pointers: xyz [n][3], owner [n] (atom index of the point's grid), w_part [n] (output).  The caller
 * multiplies with the radial and angular quadrature weights to obtain aims_grid_desc.w.
 * Limits (AIMS_ERR_UNSUPPORTED, text in aims_gpu_last_error): at most 256 atoms within r_part of any one point -- found on the
 * device; w_part of such a point is 0, the other points are valid --; the atoms' bounding box may span at most 2048 cells of
 * edge r_part along an axis and 2^26 cells in all.  The call waits for the context stream before it returns (it reads the
 * device's flag back), so an error is reported by this call, not by a later aims_gpu_synchronize.  The cell list of the atoms
 * is kept in the context for the last r_part used. */
int aims_gpu_partition_weights(aims_gpu_ctx *ctx, int64_t n, const double *xyz, const int32_t *owner, double r_part,
                               double *w_part);

/* The same weights for a caller that must not allocate device memory.  Who that is: a rank that shares its GPU with other
 * MPI tasks through MPS (how the paper runs) under a per-client memory limit its own pools have already used
 * up; a host program whose caching allocator (torch's, an MD driver's) holds all free HBM, so that a raw cudaMalloc fails
 * although the program still has room; and a loop that cannot afford the device-wide stall of cudaMalloc / cudaFree.  For
 * them every other call here is out of reach: aims_gpu_create allocates, and aims_gpu_partition_weights needs a context
 * and grows a buffer.  The weights come before the context in any case (they go into aims_grid_desc.w), so this call
 * takes no context: the atoms are passed directly and the caller still owns every input and output array.
 *
 * The scratch the kernel needs next to them -- the cell list of the atoms, the device copy of their positions, one flag
 * word -- lives in a fixed array inside the library, AIMS_NOALLOC_SCRATCH_BYTES (about 1.5 MB) of device memory that EVERY
 * GPU which loads the library holds until the process exits, whether this call is used or not.  That fixes the sizes:
 *   n_atoms <= AIMS_NOALLOC_MAX_ATOMS, and the cells of edge r_part spanned by the atoms' bounding box <= AIMS_NOALLOC_MAX_CELLS;
 * anything larger returns AIMS_ERR_UNSUPPORTED and says which limit in err_text; nothing has been enqueued then.  A point
 * with more than 256 atoms within r_part also returns AIMS_ERR_UNSUPPORTED (found on the device; w_part of such points is 0,
 * the others are valid).  The call makes no cudaMalloc / cudaFree and uses no library routine that allocates device memory;
 * on the host it builds the cell list in ordinary heap vectors.
 *
 * Arguments.  HOST: atom_xyz [n_atoms][3] (NULL only if n_atoms == 0; read during the call); err_text NULL or a buffer of
 * err_capacity bytes that receives a NUL-terminated message on failure ("" on success).  DEVICE, on `device`: xyz [n][3],
 * owner [n], w_part [n] (output).  Same definition, same kernel and the same results as aims_gpu_partition_weights.
 * Enqueued on `cuda_stream` of `device`; the call waits for that stream before it returns (it reads the flag word back).
 *
 * Sharing.  All calls on one device use the one array, and it keeps what the last call wrote: each call overwrites the
 * part it reads and clears the flag word first, so calls one after another need no care.  Two calls that are in flight on
 * the same GPU at once (two host threads, each on its own stream) overwrite each other's cell list -- a race the library
 * does not guard against; keep such calls apart yourself.  Other devices, and other processes, have their own copy.
 *
 * First call on a device.  It looks up where the array lives on that device (once per device and process, with that device
 * made current) and keeps the address.  Make this first call before you begin any stream capture on that device. */
#define AIMS_NOALLOC_MAX_ATOMS 16384
#define AIMS_NOALLOC_MAX_CELLS 262144
#define AIMS_NOALLOC_SCRATCH_BYTES (4 * (AIMS_NOALLOC_MAX_CELLS + 64) + 4 * AIMS_NOALLOC_MAX_ATOMS + 24 * AIMS_NOALLOC_MAX_ATOMS + 256)
int aims_gpu_partition_weights_noalloc(int device, void *cuda_stream, int32_t n_atoms, const double *atom_xyz, int64_t n,
                                       const double *xyz, const int32_t *owner, double r_part, double *w_part,
                                       char *err_text, int32_t err_capacity);

/* Row f3 of SURVEY.md 8(f): periodic boundary conditions.  The real-space matrix h^uc of Eq. 12 runs over
 * the N_rs functions of the cell atoms AND their periodic images that reach into the cell; the caller passes all of them as
 * atoms (the cell's own atoms first) with the grid points mapped back into the cell at T = 0 (L113-115), and
 * aims_gpu_integrate_hamiltonian / aims_gpu_update_density run unchanged ("the exact same real-space integration code").
 * This call forms the Bloch sums of Eq. 7 inserted into Eq. 11 (L115):
 *   out[i][j] (+)= sum_{I image of i} sum_{J image of j} e^{i k.(T_J - T_I)} H[I][J],   i, j = functions of the cell atoms.
 * H_values: DEVICE [n_values] (h^uc or s^uc, upper blocks, symmetric).  HOST inputs: atom_home [n_atoms] (index < n_home of the
 * cell atom an atom is an image of; atoms 0..n_home-1 are the cell's own, with atom_T = 0), atom_T [n_atoms][3] lattice
 * translations, kpt [3] (rad / Angstrom).  DEVICE outputs out_re, out_im: dense row-major [n_hb][n_hb], n_hb = functions of
 * the cell atoms.  accumulate == 0: zeroed first.  Synchronises the context stream before returning. */
int aims_gpu_bloch_fold(aims_gpu_ctx *ctx, const double *H_values, const int32_t *atom_home, const double *atom_T,
                        int32_t n_home, const double *kpt, double *out_re, double *out_im, int accumulate);

/* Row f3, geometry.  The paper says which functions enter h^uc of Eq. 12 ("all N_rs basis functions that are
 * non-zero on the unit cell", centred in the cell or in its periodic images, L109-113) and that "each integration point r is mapped
 * back to its periodic image within the unit cell at T = (0,0,0)" (L113-115), but states neither rule; reading P23:
 *
 * aims_gpu_periodic_images.  lattice: HOST [3][3], rows a_1, a_2, a_3; frac: HOST [n_home][3] fractional coordinates of the cell
 * atoms, each in [0, 1) (anything else, NaN included, returns AIMS_ERR_INVALID_ARG: the enumeration box is sized for atoms inside the cell).  With h_i = V / |a_j x a_k| (height of the cell along the i-th reciprocal direction) and delta_i = reach / h_i, the
 * periodic atom (a, n) = cell atom a translated by the integer vector n is kept iff -delta_i < frac[a][i] + n_i < 1 + delta_i for
 * i = 1, 2, 3 -- a parallelepiped containing every point within `reach` of the cell, i.e. a superset of the atoms whose functions
 * (cutoff <= reach) are non-zero somewhere in the cell; the per-batch culling of aims_gpu_eval_basis drops the rest.  Order: the
 * cell's own atoms first (n = 0, ascending a), then ascending (n_1, n_2, n_3, a).  HOST outputs: atom_home [capacity],
 * atom_n [capacity][3], *n_atoms = number of periodic atoms.  capacity == 0 is a size query (returns AIMS_OK); 0 < capacity <
 * *n_atoms returns AIMS_ERR_INVALID_ARG with *n_atoms set.  Runs on the host (a few thousand atoms); no context, no device.
 * The caller forms atom_xyz = (frac[home] + n) . lattice and atom_T = n . lattice for aims_gpu_create / aims_gpu_bloch_fold. */
int aims_gpu_periodic_images(const double *lattice, int32_t n_home, const double *frac, double reach, int32_t *atom_home,
                             int32_t *atom_n, int64_t capacity, int64_t *n_atoms);

/* aims_gpu_wrap_points.  xyz: DEVICE [n_points][3], in place: f = r A^-1 (A = lattice rows; A^-1 by the cofactor formula,
 * determinant along the first row, computed on the host), f <- f - floor(f) (and f <- 0 where that difference rounds to 1.0, so
 * that f lies in [0, 1) also for a point a hair below a cell face), r <- f A; every product and sum separately rounded
 * (IEEE RN, no FMA), sums left to right, so that exactly one result is correct.  lattice: HOST [3][3].  Enqueued on `cuda_stream` of
 * `device`; asynchronous.  A singular lattice returns AIMS_ERR_INVALID_ARG. */
int aims_gpu_wrap_points(int device, void *cuda_stream, const double *lattice, int64_t n_points, double *xyz);

/* Row f4 of SURVEY.md 8(f): the grid-adapted cut-plane batching of PAPER.md L210-218 on the GPU.  The paper cites "Algorithm 3 of
 * [37]" without stating it; reading P12 fixes a deterministic recursive bisection: a set of n points is a batch if
 * n <= max_batch_points; otherwise, with nb = ceil(n / max_batch_points), the n_left = round(floor(nb/2) n / nb) points smallest in
 * (coordinate along the axis of largest extent -- ties to x, then y --, original index) form the left child and the rest the
 * right child; batches are emitted depth-first and keep the order of their parent's sort.  Exactly one result is correct.
 * No context is needed (batching precedes aims_gpu_create).  xyz: DEVICE [n_points][3]; order: DEVICE output [n_points],
 * order[k] = original index of the point at position k of the batched grid; batch_ptr: HOST output, n_batches + 1 entries
 * (capacity batch_ptr_capacity >= 2 ceil(n_points / max_batch_points) + 2 always suffices); n_batches: HOST output.
 * Runs on `cuda_stream` of `device` and synchronises it before returning.  n_points < 2^31. */
int aims_gpu_batch_points(int device, void *cuda_stream, int64_t n_points, const double *xyz, int32_t max_batch_points,
                          int64_t *order, int64_t *batch_ptr, int64_t batch_ptr_capacity, int32_t *n_batches);

/* Bitwise-reproducible H (PAPER.md L231 leaves the order of the batch sums free, it does not forbid a
 * fixed one).  enable != 0: aims_gpu_integrate_hamiltonian[_ks] and aims_gpu_add_tau_matrix add every batch's contribution
 * to H in ascending batch order ("ordered scatter": a tile of batch b waits until all tiles of the batches before b have
 * added), so that two runs with the same inputs, batch range, accumulate history and workspace size give bit-identical
 * H_values.  Default 0: contributions are added with floating-point reductions in arrival order (reruns agree to rounding).
 * n, grad n and hess n are reduced without atomics and are bitwise reproducible in either mode; F is not. */
int aims_gpu_set_deterministic(aims_gpu_ctx *ctx, int enable);

/* Synchronise the context stream and report anything the device flagged since the last check: an asynchronous CUDA
 * fault (AIMS_ERR_CUDA) or a failed device-side capacity / consistency check (AIMS_ERR_UNSUPPORTED). */
int aims_gpu_synchronize(aims_gpu_ctx *ctx);

/* Static structure found at creation (HOST outputs, any may be NULL): sum and max over all batches of |nnz(B)|,
 * max number of active atoms, algorithmic flops of one full H pass (GGA: 2*sum n_p nnz^2; LDA: sum n_p nnz (nnz+1))
 * and of one density pass (2*sum n_p nnz^2). */
int aims_gpu_stats(aims_gpu_ctx *ctx, int64_t *sum_nnz, int32_t *max_nnz, int32_t *max_active_atoms,
                   double *flops_h_lda, double *flops_h_gga, double *flops_density);

/* |nnz(B)| of every batch as found at creation (HOST output, [n_batches]); used to balance batch ranges over GPUs. */
int aims_gpu_batch_nnz(aims_gpu_ctx *ctx, int32_t *nnz);

/* ===================================================== diagnostics =====================================================
 * Nothing below is needed to compute anything; bench.py and the profiles use it. */

/* Compile-time switches this library was built with: "" for the product build (the only one whose results are H, n, ...), else
 * the -D list of a measurement ("probe") build of paper_1912_06636_b200/build.py --define ... --tag ..., some of which switch
 * parts of the arithmetic off on purpose.  Static string.  The Python binding refuses a library that reports switches unless
 * the caller asks for it by path and says so (load_library(path, allow_probe=True); bench.py --lib). */
const char *aims_gpu_build_flags(void);

/* Per-kernel device timing for bench.py's roofline: when enabled, every kernel launch of this context is bracketed by
 * CUDA events on the context stream.  aims_gpu_timing_enable synchronises, clears what was recorded and switches
 * recording on (enable != 0) or off.  aims_gpu_timing_read synchronises and returns, since the last enable/read, the
 * summed device milliseconds ms[6] and launch counts launches[6] (HOST outputs) of
 *   [0] k_cull  [1] k_eval  [2] k_hamiltonian  [3] k_density  [4] other  [5] k_forces / k_density_hessian. */
int aims_gpu_timing_enable(aims_gpu_ctx *ctx, int enable);
int aims_gpu_timing_read(aims_gpu_ctx *ctx, double *ms, int64_t *launches);

/* Number of kernels this context has launched since creation (for bench.py's gpu_launches). */
int64_t aims_gpu_launch_count(const aims_gpu_ctx *ctx);

/* FP64 tensor-pipe (DMMA.8x8x4) peak probe: runs a dependency-free mma.sync.m8n8k4.f64 chain on every SM for about
 * `ms_target` milliseconds on the context stream and returns the achieved TFLOP/s in *tflops (HOST output).
 * Used by bench.py as the measured FP64 roofline denominator. */
int aims_gpu_fp64_peak(aims_gpu_ctx *ctx, double ms_target, double *tflops);

/* DMMA operand-pattern probe behind the K-loop design of the contraction kernels: warps_per_sm warps
 * per SM (1..16) each run 16 DMMA.8x8x4 per step on a 32x32 accumulator block with
 *   variant 1: operands in registers;  2: the step's 8 fragments loaded from shared memory, then its DMMAs;
 *   variant 3: the loads of the next step issued before the DMMAs of the current one;
 * variants 4..9 (warps_per_sm 1..20) run the K-step body of the kernels on a (WA x WB) block of 8x8 accumulator tiles:
 *   4, 5, 6, 9: fragments reloaded in place, blocks 4x4, 4x3, 3x3, 2x2;  7, 8: second fragment register set, blocks 4x4, 4x3;
 *   10, 11: the in-place 4x3 step inside the kernels' control flow (trip counts from global memory, stage loop around a step loop);
 *   11 with the four steps of a stage unrolled into one block.
 * Returns the achieved TFLOP/s in *tflops (HOST output).  Diagnostic only. */
int aims_gpu_dmma_probe(aims_gpu_ctx *ctx, int variant, int warps_per_sm, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* AIMS_GPU_H */
