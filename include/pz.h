/*
 * pz.h -- C ABI of the B200-native Poisson + wall-normal Helmholtz hot path of
 * arxiv/paper_2502_06296 (Diez, Peeters, Costa: pencil-distributed finite-difference
 * solver for turbulent wall flows).  Citations are PAPER.md:<line>.
 *
 * Everything behind this boundary is hand-written CUDA for sm_100a in FP64.  There is no
 * CPU fallback: without a CUDA device every compute entry point returns PZ_ECUDA.
 *
 * Conventions
 *   - Fields are compact C-order arrays p[k][j][i] of nx*ny*nz doubles, x (i) fastest,
 *     z (k) slowest, no ghost cells.  Element offsets are 64-bit.
 *   - "device" pointers are CUDA device addresses, "host" pointers are ordinary host
 *     addresses (pinned memory is faster for the *_host calls but not required).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - All solves are IN PLACE ("only the array d' is modified in-place"),
 *     asynchronous on `stream`, allocate nothing, never synchronise the host, use no
 *     atomics (bitwise run-to-run deterministic) and can be captured into a CUDA graph.
 *   - The caller owns every array it passes; zc/zf are copied at plan creation.  The plan
 *     owns its device tables and workspace until poisson_plan_destroy.
 *   - Every function returns a pz_status; on failure pz_last_error() holds a message
 *     (thread-local) and no output array has a defined value.
 *
 * Grid: uniform spacing lx/nx, ly/ny in the periodic directions; wall-normal cell faces
 * zf[0..nz] (strictly increasing) and cell centres zc[0..nz-1] with zf[k] < zc[k] < zf[k+1]
 * (staggered grid, uniform x,y, non-uniform z, second-order differences).
 *   dzf_k = zf[k+1]-zf[k], dzc_k = zc[k+1]-zc[k],
 *   A_k = 1/(dzf_k dzc_{k-1}) (A_0 = 0),  C_k = 1/(dzf_k dzc_k) (C_{nz-1} = 0).
 */
#ifndef PZ_H
#define PZ_H

#if defined(__GNUC__)
#define PZ_API __attribute__((visibility("default")))
#else
#define PZ_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pz_plan pz_plan; /* opaque */

enum pz_status {
    PZ_OK = 0,
    PZ_EINVAL = 1,       /* null pointer, non-positive size, non-monotone grid, a < 0, ... */
    PZ_EUNSUPPORTED = 2, /* nx or ny outside the supported lengths, nz < 4, unknown bc/option */
    PZ_ENOMEM = 3,       /* host or device allocation failed */
    PZ_ECUDA = 4,        /* CUDA runtime error (message in pz_last_error) */
    PZ_ENOTSETUP = 5     /* helmholtz_z_solve before helmholtz_z_setup */
};

/* Boundary conditions of the Poisson solve ("Fourier / cosine / sine" expansions,
 * "multiple combinations of boundary conditions"), one code per direction, combined with PZ_BC:
 *   x, y:  PZ_PERIODIC, PZ_NEUMANN (zero gradient at both ends: cosine transform) or PZ_DIRICHLET
 *          (zero value at both end FACES: sine transform);
 *   z:     PZ_Z_NN (zero wall-normal gradient at both walls), PZ_Z_DD (zero value at both wall
 *          faces), PZ_Z_ND (gradient at the bottom, value at the top), PZ_Z_DN.
 * bc = 0 is the hot path of BASELINE.json: periodic x, y, Neumann walls.  Wherever no direction has
 * a constant eigenvector (any Dirichlet end) the problem is non-singular and nothing is pinned.
 * The Helmholtz solves keep u = 0 on the wall faces whatever bc; helmholtz3d_*, the z-slab plans
 * and the pressure-correction calls need bc = 0. */
enum pz_bc_dir { PZ_PERIODIC = 0, PZ_NEUMANN = 1, PZ_DIRICHLET = 2 };
enum pz_bc_z { PZ_Z_NN = 0, PZ_Z_DD = 1, PZ_Z_ND = 2, PZ_Z_DN = 3 };
#define PZ_BC(bcx, bcy, bcz) ((bcx) + 4 * (bcy) + 16 * (bcz))
enum pz_bc { PZ_BC_PERIODIC_XY_NEUMANN_P_DIRICHLET_U = 0 };

/*
 * Plan / pre-processing (PAPER.md:199 "only once as an initialization step", :338
 * "inexpensive operation ... during the initialization").  Builds on the host and uploads:
 * the z-metric tables A_k, C_k, dzf_k; the modified wavenumbers lambda_x, lambda_y
 * re-ordered for the packed half-complex layout; the FFT
 * twiddle tables.  No field-sized device memory is allocated by the default solver variants.
 *   out    receives the plan (host pointer to host pointer)
 *   zc,zf  host arrays of nz and nz+1 doubles
 * Errors: PZ_EINVAL, PZ_EUNSUPPORTED, PZ_ENOMEM, PZ_ECUDA.
 */
PZ_API int poisson_plan_create(pz_plan **out, int nx, int ny, int nz, double lx, double ly,
                        const double *zc, const double *zf, int bc);

/*
 * Pressure Poisson solve, Eq. (4)/(12), steps 2-8 of PAPER.md:124-131:
 * real FFT along x, FFT along y, one tridiagonal solve along z per (kx,ky) with the
 * eigenvalue lambda_x(i)+lambda_y(j) added to the diagonal -(A_k+C_k) (Neumann walls),
 * inverse FFTs, 1/(nx ny) scaling.  On entry p = right-hand side f, on return p = phi with
 *   (L_h phi) = f   and   sum_ijk dzf_k phi_ijk = 0   (the singular (0,0) mode is solved with
 * its last wall-normal equation replaced by the gauge and carries zero volume mean).
 * f must be compatible (sum_ijk dzf_k f_ijk = 0); this is not checked.
 *   p  device, nx*ny*nz doubles, 16-byte aligned, in place.
 */
PZ_API int poisson_solve(pz_plan *plan, double *p, void *stream);

/*
 * ONE Poisson problem spread over several ranks (GPUs) by z-slabs: the paper's parallel tridiagonal
 * solver, PAPER.md:120-135 (steps 1-8 of section 2.2.3) and :139-155, with GPUs for its "MPI tasks".
 * Rank `slab` of `n_slabs` owns the planes [kbounds[slab], kbounds[slab+1]) of the global grid of nz
 * planes (kbounds: host, n_slabs + 1 ints, from 0 to nz, at least 3 and at most 1024 planes per slab,
 * PAPER.md:284; n_slabs <= 16); x and y transforms are plane-local.  zc, zf describe the GLOBAL grid.
 * Plan creation also computes, on the device, the right-hand-side-independent coefficients of the
 * reduced boundary systems of ALL slabs ("only once as an initialization step"; every
 * rank computes them itself, so creating the plans needs no communication).
 *
 * A solve is two calls around ONE collective that the caller performs (e.g. NCCL all-gather):
 *   poisson_solve_reduce   p (device, this rank's nx*ny*nk doubles, in place): forward transforms,
 *                          slab-local reduction; writes this rank's boundary values into
 *                          boundary_out (device, poisson_slab_boundary_doubles(plan) doubles:
 *                          2 nx ny values "packed" as in PAPER.md:127 plus the slab's rows of the
 *                          singular (0,0) column).
 *   [all-gather boundary_out of every rank, in rank order, into boundary_all]
 *   poisson_solve_finish   solves the reduced systems of size 2 n_slabs for every column
 *                          (redundantly on every rank), reconstructs the slab and
 *                          applies the inverse transforms: p holds this rank's planes of phi, the
 *                          same solution poisson_solve gives on one GPU (zero volume mean).
 * Errors: PZ_EINVAL (bad bounds, NULL, not a slab plan), PZ_EUNSUPPORTED (slab thickness), PZ_ENOMEM,
 * PZ_ECUDA.  poisson_solve, helmholtz_* and helmholtz3d_* refuse a slab plan.
 */
PZ_API int poisson_slab_plan_create(pz_plan **out, int nx, int ny, int nz, double lx, double ly,
                             const double *zc, const double *zf, int bc, int n_slabs, int slab,
                             const int *kbounds);
PZ_API long long poisson_slab_boundary_doubles(const pz_plan *plan);
PZ_API int poisson_solve_reduce(pz_plan *plan, double *p, double *boundary_out, void *stream);
PZ_API int poisson_solve_finish(pz_plan *plan, double *p, const double *boundary_all, void *stream);

/*
 * The same solve with the exchange done by the kernels themselves over peer memory (NVLink /
 * NVSwitch) instead of a collective: every rank owns a gathered buffer boundary_all (n_slabs *
 * poisson_slab_boundary_doubles doubles) and a flag array (n_slabs 64-bit integers, zero-initialised)
 * that ALL ranks of the node can address (peer-mapped / symmetric memory; the caller obtains the
 * pointers, e.g. torch.distributed._symmetric_memory).
 *   poisson_solve_reduce_push   forward transforms and reduction; the reduction kernel stores this
 *                               rank's block straight into its slot of EVERY rank's boundary_all
 *                               (boundary_all_of_rank[r], host array of n_slabs device pointers),
 *                               then releases flags_of_rank[r][slab] = epoch at system scope.
 *   poisson_solve_finish_wait   waits on the device until all n_slabs entries of this rank's own
 *                               flag array have reached epoch, then poisson_solve_finish.
 * epoch must grow by one per solve.  Every rank must enqueue its push before its wait (the wait
 * spins on the device); the buffers of solve e must not be rewritten before every rank has
 * finished solve e (two buffer sets alternate in sharded.SlabPoisson).
 */
PZ_API int poisson_solve_reduce_push(pz_plan *plan, double *p, double *const *boundary_all_of_rank,
                                     long long *const *flags_of_rank, long long epoch, void *stream);
PZ_API int poisson_solve_finish_wait(pz_plan *plan, double *p, const double *boundary_all, const long long *flags,
                                     long long epoch, void *stream);

/*
 * Wall-normal implicit diffusion, Eq. (11), with the paper's split of the
 * cyclic-reduction solver into pre-processing and runtime (Algorithm 2).
 *
 * helmholtz_z_setup: pre-processing for (I - a L_z), a = gamma_k nu dt / 2 >= 0.  Computes the
 * k-only coefficient sub-arrays of Algorithm 2 Step 1 for every sub-domain, and the per-level
 * multipliers of the cyclic reduction of the boundary system, on the host (O(nz) work), and
 * uploads them into a table set that no solve still in flight and no captured CUDA graph reads.
 * May be called once per Runge-Kutta sub-step ("time-dependent").
 * CUDA graphs: a helmholtz_z_solve / _solve_n / helmholtz_z_step captured into a graph keeps the
 * table set (and so the coefficient a) that was current at capture time; that set stays untouched
 * until poisson_plan_destroy, so replays remain valid across any number of later set-ups or
 * geometry options, and solve with the captured a.  Capture after the set-up for that a.
 *
 * helmholtz_z_solve: runtime.  For every (i,j) column solves
 *   u_k - a [A_k (u_{k-1}-u_k) + C_k (u_{k+1}-u_k) - W_k u_k] = r_k,
 * W_k = 0 except W_0 = 1/(dzf_0 (zc_0-zf_0)), W_{nz-1} = 1/(dzf_{nz-1} (zf_nz-zc_{nz-1}))
 * (u = 0 on the wall faces), touching only the right-hand side (Algorithm 2 Steps 2-4).
 *   u  device, nx*ny*nz doubles, in place: on entry r, on return u.
 * helmholtz_z_solve_n applies the same operator to n fields (the three velocity components).
 * Errors: PZ_ENOTSETUP before the first setup; PZ_EINVAL for a < 0 or null pointers;
 * PZ_EUNSUPPORTED from the set-up for nz > 3584 (a column chunk no longer fits shared memory).
 */
PZ_API int helmholtz_z_setup(pz_plan *plan, double a);
PZ_API int helmholtz_z_solve(pz_plan *plan, double *u, void *stream);
PZ_API int helmholtz_z_solve_n(pz_plan *plan, double *const *u, int n, void *stream);

/*
 * The same solve for the wall-normal velocity component w, which lives on the z FACES of the
 * staggered grid: w[k] on the face zf[k+1], k = 0..nz-1; the bottom wall face zf[0]
 * carries w = 0 and is not stored, the top wall face is row nz-1 and keeps its value.  For
 * k = 0..nz-2 (w_{-1} = w_{nz-1} = 0 in the operator):
 *   w_k - a [ (w_{k+1} - w_k)/dzf_{k+1} - (w_k - w_{k-1})/dzf_k ] / dzc_k = r_k.
 * Its coefficient tables are independent of those of helmholtz_z_setup: a time step sets up both
 * and solves u, v with helmholtz_z_solve_n and w with helmholtz_w_solve.  Same kernels, same
 * CUDA-graph rules.  Errors as helmholtz_z_setup / helmholtz_z_solve.
 */
PZ_API int helmholtz_w_setup(pz_plan *plan, double a);
PZ_API int helmholtz_w_solve(pz_plan *plan, double *w, void *stream);

/*
 * The whole of Eq. (11):  u* - a L_z u* = u** - a L_z u^k  with the a of the last
 * helmholtz_z_setup.  helmholtz_z_rhs overwrites ustar2 (on entry u**) with the right-hand side
 * u** - a L_z u^k, L_z the operator above; helmholtz_z_step does that and then helmholtz_z_solve:
 * on return ustar2 holds u*.  uk is only read.  Both device, nx*ny*nz doubles, 16-byte aligned.
 * Errors: PZ_ENOTSETUP before the first setup; PZ_EINVAL for null or misaligned pointers.
 */
PZ_API int helmholtz_z_rhs(pz_plan *plan, double *ustar2, const double *uk, void *stream);
PZ_API int helmholtz_z_step(pz_plan *plan, double *ustar2, const double *uk, void *stream);

/*
 * Fully implicit diffusion, Eq. (8), PAPER.md:63-72 ("a Helmholtz equation for the prediction
 * velocity, implicit in the three spatial directions", solved "using the fast direct methods" of
 * the Poisson solve): for a = gamma_k nu dt / 2 >= 0 solves, in place,
 *   (I - a L_h) u = r,   L_h = the 7-point Laplacian of poisson_solve in x, y (periodic) and
 *   A_k (u_{k-1}-u_k) + C_k (u_{k+1}-u_k) - W_k u_k in z (u = 0 on the wall faces, W as above).
 * Same pipeline as poisson_solve: transforms along x and y, one tridiagonal solve per (kx,ky)
 * with diagonal 1 + a (A_k + C_k + W_k - lambda_x - lambda_y), inverse transforms.  The systems
 * are non-singular for every mode (no pinned column).  helmholtz3d_setup only records a (the
 * coefficient tables are scaled inside the kernel), so it may be called between any two solves.
 *   u  device, nx*ny*nz doubles, 16-byte aligned, in place.  Above 1024 planes the z stage runs as a
 *      thread-per-column sweep (one field of workspace, allocated on first use).
 * Errors: PZ_ENOTSETUP before the first setup; PZ_EINVAL for a < 0 or null pointers;
 * PZ_EUNSUPPORTED on plans with bc != 0 or z-slab plans.
 */
PZ_API int helmholtz3d_setup(pz_plan *plan, double a);
PZ_API int helmholtz3d_solve(pz_plan *plan, double *u, void *stream);

/*
 * The steps either side of the Poisson solve in the pressure-correction scheme,
 * on the staggered grid: u[k][j][i] on the x-face between cells i and i+1, v on the y-face between
 * j and j+1 (periodic), w on the z-face zf[k+1] (the bottom wall face carries w = 0 and is not
 * stored; w[nz-1] is the top wall face and should be 0), p and Phi at cell centres.
 *   pz_divergence_rhs      rhs = D u* / (gamma dt), Eq. (4):
 *                          (u_i-u_{i-1})/dx + (v_j-v_{j-1})/dy + (w_k-w_{k-1})/dzf_k, times inv_gdt
 *   pz_project             u -= gamma dt G Phi (Eq. 5), p += Phi (Eq. 6); the top wall face of w
 *                          is left untouched (zero wall-normal gradient of Phi)
 *   pz_pressure_correction both around poisson_solve: work <- rhs, solved in place, then the
 *                          correction; afterwards D u = 0 to rounding (D G is the operator of
 *                          poisson_solve exactly).  work: device, nx*ny*nz doubles, holds Phi on return.
 * All fields: device, nx*ny*nz doubles, 16-byte aligned; in place where written.
 */
PZ_API int pz_divergence_rhs(pz_plan *plan, const double *u, const double *v, const double *w, double *rhs,
                             double inv_gdt, void *stream);
PZ_API int pz_project(pz_plan *plan, double *u, double *v, double *w, double *p, const double *phi, double gdt,
                      void *stream);
PZ_API int pz_pressure_correction(pz_plan *plan, double *u, double *v, double *w, double *p, double *work, double gdt,
                                  void *stream);

/*
 * End-to-end variants with HOST buffers: copy host -> device workspace (owned by the plan,
 * allocated on first use: nx*ny*nz doubles), solve, copy back, all asynchronously on
 * `stream`.  The host buffer must stay valid until the stream has been synchronised.
 */
PZ_API int poisson_solve_host(pz_plan *plan, double *p_host, void *stream);
PZ_API int helmholtz_z_solve_host(pz_plan *plan, double *u_host, void *stream);

/*
 * One time step's worth of solves on HOST buffers, pipelined: the Poisson field p_host (may be
 * NULL) and the n_u Helmholtz fields u_host[0..n_u-1] go through three device staging fields
 * (owned by the plan, allocated on first use) so that the upload of field f+1, the solve of field
 * f and the download of field f-1 overlap (two internal copy streams; the PCIe link is full
 * duplex).  Ordered after prior work on `stream`; when `stream` has been synchronised every
 * host buffer holds its solution.  Pinned host memory is needed for the copies to overlap.
 * Errors: as the single-field calls; PZ_ENOTSETUP if n_u > 0 before helmholtz_z_setup.
 */
PZ_API int pz_solve_host_batch(pz_plan *plan, double *p_host, double *const *u_host, int n_u, void *stream);

/* Step a3 alone (the z tridiagonal solves of Eq. 12; steps 4-6 of PAPER.md:127-129)
 * for callers that may not allocate: code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc.  The thread-per-column sweep (z-solve variant 0) stages its
 * multipliers C_k / p_k in a workspace of N doubles, which the ordinary path allocates on first use;
 * here that workspace is a file-scope device array of the library of
 *     PZ_NOALLOC_MAX_POINTS = 2^21 doubles (16 MiB),
 * which every GPU that loads libpz_b200.so holds until the process exits.
 *   plan    an ordinary plan (poisson_plan_create; not a z-slab plan), any boundary-condition code
 *   p       device, N = nx ny nz doubles, the field AFTER the forward transforms (packed spectral
 *           layout, as PZ_STAGE_Z_SOLVE of pz_poisson_stage takes it); solved in place
 *   stream  cudaStream_t or NULL
 * The call itself calls no cudaMalloc / cudaFree and no allocating library routine (the first call on
 * a device looks the array's address up with cudaGetSymbolAddress).  The plan's device must be
 * current.  PZ_EUNSUPPORTED if N > PZ_NOALLOC_MAX_POINTS (nothing is launched), PZ_EINVAL for NULL /
 * misaligned pointers, a z-slab plan or another current device, PZ_ECUDA for CUDA errors.
 * ALL calls, from every plan and stream of the process, share the one array: calls that overlap on
 * the GPU race and give wrong results -- keep them on one stream or order them with events.  Nothing
 * in the array needs to start at zero (every entry is written by the forward sweep before the
 * backward sweep reads it), so the contents a previous call leaves behind are harmless.
 * Result: bitwise the one of pz_poisson_stage(plan, p, PZ_STAGE_Z_SOLVE) with zsolve_variant = 0. */
#define PZ_NOALLOC_MAX_POINTS (1LL << 21)
PZ_API int poisson_zsolve_noalloc(pz_plan *plan, double *p, void *stream);

/* Frees every device and host resource of the plan.  NULL is accepted. */
PZ_API int poisson_plan_destroy(pz_plan *plan);

/* Message of the last failure on the calling thread ("" if none). */
PZ_API const char *pz_last_error(void);

/* ------------------------------------------------------------------ diagnostics
 * Used by the tests, the benchmark and the profiles; not needed by a solver user. */

/* Stages of poisson_solve, runnable one at a time on a device field (in place). */
enum pz_stage {
    PZ_STAGE_FFT_X_FWD = 0, /* a1: R2C along x into the packed layout                     */
    PZ_STAGE_FFT_Y_FWD = 1, /* a2: FFT along y of the packed complex pairs                */
    PZ_STAGE_Z_SOLVE = 2,   /* a3: tridiagonal solves in spectral space                   */
    PZ_STAGE_FFT_Y_INV = 3, /* a4                                                         */
    PZ_STAGE_FFT_X_INV = 4, /* a5: C2R along x and 1/(nx ny) scaling                      */
    PZ_STAGE_FFT_XY_FWD = 5, /* a1+a2 by the fused kernel (nx in {256,..,2048}, ny in {256,512,1024}) */
    PZ_STAGE_FFT_XY_INV = 6  /* a4+a5 by the fused kernel                                  */
};
PZ_API int pz_poisson_stage(pz_plan *plan, double *p, int stage, void *stream);

/* Integer tuning options (kernel variants, tile widths, slab sizes).  Unknown keys or
 * unsupported values return PZ_EUNSUPPORTED and change nothing.  Keys are listed in
 * DESIGN.md ("Options"). */
PZ_API int pz_set_option(pz_plan *plan, const char *key, int value);
PZ_API int pz_get_option(const pz_plan *plan, const char *key, int *value);

/* Per-kernel device timing for the benchmark's roofline figures.  While enabled, every kernel
 * launch of this plan is bracketed by a pair of CUDA events recorded on the launching stream
 * (no host synchronisation, a few microseconds of stream time per launch).
 * pz_profile_enable(plan, 1) clears the records and starts; (plan, 0) stops.
 * pz_profile_read synchronises on the recorded events and returns, for one kernel class, the
 * summed device time in milliseconds and the number of launches.  Not capturable in a graph. */
enum pz_kernel_class {
    PZ_K_FFT_X_FWD = 0, PZ_K_FFT_Y_FWD = 1, PZ_K_PAIR0_FWD = 2, PZ_K_Z_SOLVE = 3,
    PZ_K_PAIR0_INV = 4, PZ_K_FFT_Y_INV = 5, PZ_K_FFT_X_INV = 6, PZ_K_HELMHOLTZ = 7,
    PZ_K_FFT_XY_FWD = 8, /* a1+a2 in one kernel (second trip of the plane through L2 only) */
    PZ_K_FFT_XY_INV = 9, /* a4+a5 in one kernel */
    PZ_K_DIV_RHS = 10,   /* pz_divergence_rhs */
    PZ_K_PROJECT = 11,   /* pz_project */
    PZ_K_HELM_RHS = 12,  /* helmholtz_z_rhs */
    PZ_K_COUNT = 13
};
PZ_API int pz_profile_enable(pz_plan *plan, int on);
PZ_API int pz_profile_read(pz_plan *plan, int kernel_class, double *total_ms, long long *launches);

/* Host logic of the mixed-radix transforms (paper: "in-house mixed-radix FFT"; DESIGN.md
 * section 14): the radices, first pass first, that the kernels use for a complex transform of length
 * n whose lines are stored `stride` elements apart in shared memory (1: x lines, the pairs per CTA: y
 * columns) when every thread must keep at least `min_points` points (1 = no constraint).  Writes at
 * most `cap` entries to radices (host pointer) and returns their number, 0 if n has a prime factor
 * above 7 or no factorisation meets min_points.  Needs no GPU. */
PZ_API int pz_fft_radices(int n, int min_points, int stride, int *radices, int cap);

/* Number of kernels this library has launched since it was loaded (host-side counter). */
PZ_API long long pz_launch_count(void);

/* Library version: major*10000 + minor*100 + patch. */
PZ_API int pz_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PZ_H */
