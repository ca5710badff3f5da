/* ptefit.h -- C ABI of the B200-native PTEFIT hot path (arxiv 2601.12378).
 *
 * The library runs the per-time-slice EFIT Picard iteration of PTEFIT on one GPU (sm_100a):
 *   basis J_b (Eq. 8-11) -> response R = G_P J_b (Eq. 6)
 *   -> least squares for X -> node currents J_b X -> boundary flux G_B I
 *   -> Delta* psi = -mu0 R J_phi by DST-in-Z + tridiagonal-in-R (Eq. 1, 118-120)
 *   -> axis / X-point / LCFS search and normalisation (Sec. II.D).
 * It never computes Green's functions (PAPER.md:65-79 is an offline precompute): the tables are
 * inputs of ptefit_create.  There is no CPU fallback: every entry point fails with
 * PTEFIT_ERR_CUDA when no sm_100 device is usable.
 *
 * Conventions: COCOS 7, psi is flux per radian; grid node (i, j) has
 * R_i = rmin + i dR, Z_j = zmin + j dZ and flat index n = j*nr + i (R fastest).
 * All matrices are row-major.  "real" = float (PTEFIT_FP32) or double (PTEFIT_FP64).
 */
#ifndef PTEFIT_H
#define PTEFIT_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ptefit_handle ptefit_handle; /* opaque; owns every device copy it makes */

typedef enum {
  PTEFIT_OK = 0,
  PTEFIT_ERR_INVALID_ARG = 1,
  PTEFIT_ERR_UNSUPPORTED = 2,
  PTEFIT_ERR_CUDA = 3,
  PTEFIT_ERR_NOMEM = 4
} ptefit_status;

typedef enum { PTEFIT_FP32 = 0, PTEFIT_FP64 = 1 } ptefit_precision;
/* Arithmetic of the two dense contractions (R = G_P J_b and psi_bdry = G_B I) in FP32 mode:
 * 3xTF32 = error-compensated tcgen05 tensor-core products (FP32-accurate), FFMA = plain FP32 FMA
 * (which also selects the FMA route of the Delta* solve).  Value 1 is reserved (a single-pass TF32
 * mode fails the parity tolerances, SURVEY.md hard part 2) and rejected by ptefit_create.
 * FP64 mode always uses FP64 arithmetic: DMMA (mma.sync f64) tensor-core products. */
typedef enum { PTEFIT_GEMM_3XTF32 = 0, PTEFIT_GEMM_FFMA = 2 } ptefit_gemm_mode;

/* Grid.  nz-1 must be a power of two in [8, 256] (DST length); nr in [5, 257]. */
typedef struct { int nr, nz; double rmin, rmax, zmin, zmax; } ptefit_grid;

/* Geometry.  All pointers are HOST memory, read during ptefit_create only. */
typedef struct {
  int n_meas;                     /* M: magnetic probes + flux loops (rows of Eq. 2)            */
  int n_coil;                     /* n_c: PF coils + eddy filaments (columns of G_C), <= 768     */
  const double *sigma;            /* [n_meas] 1-sigma of each channel, > 0 (fit weights 1/sigma)*/
  int n_lim;                      /* limiter polygon vertices, 1..256            */
  const double *lim_r, *lim_z;    /* [n_lim] inside the grid rectangle                          */
  const unsigned char *lim_mask;  /* [nz*nr] 1 = node may carry plasma; never an edge node      */
  const unsigned char *xpt_mask;  /* [nz*nr] 1 = node may host an X-point; NULL = lim_mask      */
  int ip_sign;                    /* +1 or -1: sign of the plasma current                       */
  double cold_rc, cold_zc, cold_a, cold_b; /* cold-start ellipse (warm_start = 0)               */
} ptefit_geometry;

/* Green's tables, HOST, FP64, row-major.  Columns of gp/gb that belong to edge nodes are ignored
 * (edge nodes never carry current).  Boundary-node order k of gb: bottom row j=0 (i=0..nr-1), top
 * row j=nz-1 (i=0..nr-1), left column i=0 (j=1..nz-2), right column i=nr-1 (j=1..nz-2). */
typedef struct {
  const double *gp;   /* [n_meas][nz*nr] response of channel m per ampere at node n (Eq. 2 G_P) */
  const double *gc;   /* [n_meas][n_coil] (Eq. 2 G_C)                                           */
  const double *gb;   /* [n_bnd][nz*nr]  flux/rad at boundary node k per ampere at node n       */
  const double *ggc;  /* [nz*nr][n_coil] flux/rad at node n per unit coil current               */
} ptefit_tables;

/* One basis term (a column of J_b, Eq. 10).  x = normalised flux.
 * kind 0: P' term, factor R dA;  kind 1: FF' term, factor (mu0/R) dA;  kind 2: vertical-shift term
 * -dI'/dZ (reading O4b; must be the last term, at most one; other fields ignored).
 * family 0 (POLY_EDGE0): x^i - x^N, 0 <= i < N <= 8.
 * family 1 (TENSION_SPLINE): cardinal tension spline phi_i(x) on `knots` (n_knots in [3,16], strictly
 *   increasing, HOST pointer read during create) with tension `tension` > 0; zero outside
 *   [knots[0], knots[n_knots-1]]; i = which cardinal function (BASELINE.json configs[4]; definition
 *   in DESIGN.md reading O4c -- not in the paper).  All spline terms of a basis must share one knot
 *   set and tension; kind must be 0 or 1. */
typedef struct {
  int kind, family;
  int i, N;
  int n_knots;
  const double *knots;
  double tension;
} ptefit_term;

typedef struct {
  int n_terms;                 /* 1..16                                                         */
  const ptefit_term *terms;    /* HOST                                                          */
  double lambda_reg;           /* Tikhonov weight in equilibrated coordinates; 0 = Eq. 6 as is  */
  double relax;                /* psi^{k+1} = psi^k + relax (psi_new - psi^k); 1 = plain Picard */
  int lsq_method;              /* 0 = normal equations + Cholesky, 1 = modified Gram-Schmidt QR
                                  (the two drivers of PAPER.md:116)                             */
  int fit_coils;               /* 1 = joint fit of the coil currents, Eq. 7:
                                  unknowns [X; I_C'], extra rows I_C' = I_C weighted 1/sigma_ic; the coil
                                  flux G_GC I_C' is recomputed every iteration; chi2 = measurement rows;
                                  needs n_terms + n_coil <= 96 and lsq_method 0                   */
  const double *sigma_ic;      /* [n_coil] HOST, 1-sigma of the measured coil currents (fit_coils) */
} ptefit_basis;

/* Option flags (ptefit_options.flags); 0 = defaults. */
#define PTEFIT_OPT_NO_GRAPH 1        /* launch the kernels directly instead of replaying a CUDA graph   */
#define PTEFIT_OPT_NO_FUSED_BASIS 2  /* materialise J_b in HBM instead of generating it in the GEMM     */
#define PTEFIT_OPT_SOLVE_FFMA 4      /* Delta* solve with FP32-FMA DSTs instead of the tcgen05 kernel   */

typedef struct {
  ptefit_precision precision;
  ptefit_gemm_mode gemm;
  int max_batch;               /* largest batch ptefit_reconstruct will be called with          */
  int flags;                   /* PTEFIT_OPT_* bit mask                                         */
  int tc_split_k;              /* split-K factor of the tensor-core contractions; 0 = automatic */
} ptefit_options;

/* Build a reconstruction handle: validates, copies the tables to the device (rounded to nearest
 * FP32 in FP32 mode), precomputes the DST/tridiagonal factors, allocates all workspaces for
 * max_batch slices.  The caller keeps ownership of everything it passes.  Synchronous.
 * On error *out = NULL and ptefit_global_error() describes the failure. */
ptefit_status ptefit_create(const ptefit_grid *grid, const ptefit_geometry *geom,
                            const ptefit_tables *tables, const ptefit_basis *basis,
                            const ptefit_options *opts, ptefit_handle **out);

/* Reconstruct `batch` independent time slices (1 <= batch <= max_batch), n_iter Picard
 * iterations each.  Every d_* pointer is caller-owned DEVICE memory; `real` per precision.
 * Asynchronous on `cuda_stream` (a cudaStream_t, NULL = default stream).  The launch sequence
 * of a (batch, n_iter, warm_start) combination is captured into a CUDA graph the first time it is
 * seen (that call instantiates the graph: it allocates and synchronises an internal stream);
 * every later call with the same combination only updates the graph's kernel arguments for the
 * pointers passed and launches it: no allocation, no host synchronisation.
 * Outputs that are NULL are skipped (d_psi, d_coeffs required).
 * Numerical failure of a slice is reported in d_status[slice] and never aborts the batch:
 * 0 ok, 1 plasma lost, 2 non-finite, 3 singular fit, 4 more than 32 X-point candidates.
 * After a failure the slice's other outputs are unspecified. */
ptefit_status ptefit_reconstruct(ptefit_handle *h, int batch,
    const void *d_b,        /* [batch][n_meas]  real: measurements b (Eq. 2)                    */
    const void *d_ic,       /* [batch][n_coil]  real: coil + eddy currents I_C                  */
    int n_iter, int warm_start, /* warm_start = 1: d_psi holds the starting flux, and the coefficients
                                   of this handle's previous call seed the vertical-shift column of the
                                   first iteration (slice q continues slice q of that call).
                                   warm_start = 2 ("continue", the streaming mode of PAPER.md:158): as 1, and
                                   d_psi still holds exactly what this handle's previous ptefit_reconstruct
                                   call (n_iter >= 1, batch >= this one) returned: the search of the starting
                                   flux and the rebuild of the vertical-shift column are skipped, because that
                                   call's last kernel left both behind.  PTEFIT_ERR_INVALID_ARG if there is no
                                   such call (or a ptefit_debug_* hook ran since); needs n_iter >= 1.      */
    void *d_psi,            /* [batch][nz][nr]  real, in/out: poloidal flux per radian          */
    void *d_coeffs,         /* [batch][n_terms] real: X of the last fit (Eq. 11)                */
    int *d_axis_ij,         /* [batch][2] (i, j) of the axis node                               */
    void *d_axis_rzpsi,     /* [batch][3] real: refined (R, Z, psi) of the axis                 */
    int *d_xpt_ij,          /* [batch][2] best X-point candidate node, (-1,-1) if none          */
    void *d_xpt_rzpsi,      /* [batch][3] real                                                  */
    void *d_psi_bnd,        /* [batch] real: LCFS flux                                          */
    int *d_limited,         /* [batch] 1 = boundary defined by a limiter vertex                 */
    void *d_chi2,           /* [batch] real: chi^2 of the last fit                              */
    int *d_status,          /* [batch]                                                          */
    void *cuda_stream);

/* Same as ptefit_reconstruct but every buffer is HOST memory (pageable or pinned): the call
 * copies inputs to the device, runs, copies every non-NULL output back and synchronises. */
ptefit_status ptefit_reconstruct_host(ptefit_handle *h, int batch,
    const void *b, const void *ic, int n_iter, int warm_start, void *psi, void *coeffs,
    int *axis_ij, void *axis_rzpsi, int *xpt_ij, void *xpt_rzpsi, void *psi_bnd, int *limited,
    void *chi2, int *status);

/* Test hooks (lock-step parity, tests/): run single stages on caller DEVICE buffers. */
/* Delta* solve: psi[batch][nz][nr] = solve(-mu0 R I/dA with edge data psi_bdry[batch][n_bnd]). */
ptefit_status ptefit_debug_gs_solve(ptefit_handle *h, int batch, const void *d_I /*[batch][nz*nr]*/,
                                    const void *d_psi_bdry, void *d_psi_out, void *cuda_stream);
/* Search: from d_psi fills the handle's internal state and writes xn[batch][nz*nr]
 * (normalised flux in the mask, -1 outside) and the search outputs as in ptefit_reconstruct. */
ptefit_status ptefit_debug_search(ptefit_handle *h, int batch, const void *d_psi, void *d_xn,
    int *d_axis_ij, void *d_axis_rzpsi, int *d_xpt_ij, void *d_xpt_rzpsi, void *d_psi_bnd,
    int *d_limited, int *d_status, void *cuda_stream);
/* Response + fit from xn: resp[batch][n_meas][n_terms], coeffs, chi2 (X_prev = d_xprev or 0). */
ptefit_status ptefit_debug_fit(ptefit_handle *h, int batch, const void *d_xn, const void *d_b,
    const void *d_ic, const void *d_xprev, void *d_resp, void *d_coeffs, void *d_chi2,
    int *d_status, void *cuda_stream);

/* Number of kernel launches the last ptefit_reconstruct enqueued (bench.py's gpu_launches). */
int ptefit_last_launch_count(const ptefit_handle *h);
/* Device time in ms of the stages of the last reconstruct call when profiling was enabled by
 * ptefit_set_profiling(h, 1): out[0..5] = setup, response, lsq, boundary, solve, search (sums
 * over iterations).  Profiling inserts events only; returns PTEFIT_ERR_INVALID_ARG if disabled.
 * Synchronises the stream. */
ptefit_status ptefit_set_profiling(ptefit_handle *h, int on);
ptefit_status ptefit_get_stage_ms(ptefit_handle *h, float out[6]);

/* NEXT-2: flux-surface post-processing of the last ptefit_reconstruct call of this handle
 * (Sec. II.E, Eq. 12, Fig. 1; readings in DESIGN.md O8).  For n_prof levels
 * x_p = (p + 1)/n_prof of the normalised flux and n_chord chords from the refined axis (angles 2 pi c/n_chord,
 * counter-clockwise) the vertex of every flux surface on every chord is found by n_bisect bisection steps
 * (the paper uses about 10) plus one linear interpolation; then Q_{mu,nu} = closed integral of
 * |grad psi|^mu R^nu dl (trapezoid rule on the vertex polygon) for the n_q <= 8 exponent pairs given,
 * q = (mu0 F / 2 pi) Q_{-1,-1} (NaN unless that pair is listed; F from f_vac and the fitted FF' polynomial),
 * and the geometry of the last level (LCFS): R_min, R_max, Z_min, Z_max, minor radius, elongation.
 * d_psi must be the flux that reconstruct call returned.  Outputs, DEVICE, real: d_Q[batch][n_prof][n_q],
 * d_q[batch][n_prof], d_geom[batch][6], d_vert[batch][n_prof][n_chord][2] (may be NULL),
 * d_status[batch] (may be NULL; 1 = slice failed or its axis lies outside the plasma).
 * Limits: n_prof * n_chord <= 12288, n_chord <= 1024.  Asynchronous on cuda_stream. */
typedef struct {
  int n_prof, n_chord, n_bisect;
  int n_q;
  const int *mu, *nu;            /* HOST [n_q] */
  double f_vac;                  /* vacuum R B_phi / mu0 in amperes (the paper's F at the boundary) */
} ptefit_profile_spec;
ptefit_status ptefit_flux_surfaces(ptefit_handle *h, int batch, const ptefit_profile_spec *spec, const void *d_psi,
                                   void *d_Q, void *d_q, void *d_geom, void *d_vert, int *d_status, void *cuda_stream);

/* Fitted coil currents I_C' of the last reconstruct call of a handle created with fit_coils = 1 (Eq. 7,
 * PAPER.md:87-93): d_out[batch][n_coil] real, DEVICE.  Asynchronous on cuda_stream. */
ptefit_status ptefit_get_coil_currents(ptefit_handle *h, int batch, void *d_out, void *cuda_stream);

/* NEXT-3: a Green's table on the GPU (Sec. II.A, Eq. 3-5; closed forms
 * with complete elliptic integrals, reading O1 of DESIGN.md).  out[k][c] = w_c g(field point k, source c)
 * per ampere in the source filament: g = flux per radian psi (Eq. 5) for a flux row (d_fld_cos == NULL,
 * or cos = sin = 0 for that row), g = cos a B_R + sin a B_Z for a probe row (Eq. 3-4).  All pointers are
 * DEVICE memory, FP64; d_src_w may be NULL (weights 1: e.g. turn counts); transpose = 1 stores out[c][k].
 * Coincident points give 0 (self terms are never needed: DESIGN.md O1).  Asynchronous on cuda_stream.
 * No handle: the tables are inputs of ptefit_create. */
ptefit_status ptefit_greens_table(int n_fld, const double *d_fld_r, const double *d_fld_z,
                                  const double *d_fld_cos, const double *d_fld_sin,
                                  int n_src, const double *d_src_r, const double *d_src_z,
                                  const double *d_src_w, double *d_out, int transpose, void *cuda_stream);

/* Allocation-free Delta* solve (Eq. 1; Sec. II.C), for callers that must not
 * allocate (CUDA graph capture, serving loops): the same operation as ptefit_debug_gs_solve,
 *   psi[batch][nz][nr] = solve(-mu0 R I / dA with edge data psi_bdry[batch][n_bnd]),
 * on the FP64 DMMA route (transposed right-hand side, DST in Z as a tensor-core product, FP64 Thomas in R,
 * inverse DST, transpose back) with ALL of that route's workspace -- three transposed maps and the Thomas
 * forward-sweep values, batch * (nr-2) * (3 * ld + nz-2) doubles, ld = nz-2 rounded up to even -- in one
 * file-scope __device__ array of PTEFIT_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds
 * until exit.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine (the first
 * call on a device resolves the array's device address with cudaGetSymbolAddress, which allocates nothing).
 * h: an FP64 handle whose contractions are not FFMA (it supplies the DST matrix and the tridiagonal factors,
 * which were copied at ptefit_create); the device of h must be current.  d_I[batch][nz*nr], d_psi_bdry and
 * d_psi are caller-owned DEVICE memory, FP64.  Asynchronous on cuda_stream.
 * Errors: PTEFIT_ERR_UNSUPPORTED for an FP32 / FFMA handle; PTEFIT_ERR_INVALID_ARG with a message that names
 * the need and the limit when the workspace of `batch` slices exceeds PTEFIT_NOALLOC_SCRATCH_BYTES (the limit
 * is 65 slices at 65x65, 16 at 129x129, 4 at 257x257) -- nothing is launched then.
 * The array is shared by every call, every handle and every stream of the process on that GPU and keeps the
 * last call's contents; the call clears the part it uses first.  Calls that overlap on the GPU (different
 * streams, or the same call replayed concurrently from a graph) race on it: serialise them. */
#define PTEFIT_NOALLOC_SCRATCH_BYTES (8u << 20)
ptefit_status ptefit_gs_solve_noalloc(ptefit_handle *h, int batch, const double *d_I, const double *d_psi_bdry,
                                      double *d_psi, void *cuda_stream);

void ptefit_destroy(ptefit_handle *h);
const char *ptefit_last_error(const ptefit_handle *h);
const char *ptefit_global_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PTEFIT_H */
