/*
 * snap.h — C ABI of the B200-native batched constraint projection (SNAP-FM hot path,
 * arxiv/paper_2607_00095).
 *
 *     u* = argmin_u 1/2 ||u - u_hat||^2   s.t.  h(u) = 0        (Eq. 2; Eq. 4)
 *
 * solved per sample by Gauss-Newton / Newton-KKT iterations (Eq. 5, Eq. 24 L468 with
 * W = I): each iteration evaluates the discretised-PDE residual h and its stencil-local Jacobian J
 * (PAPER.md L98-104), solves the Schur form (J J^T) lam+ = h - J (u - u_hat) of the KKT system
 * (block diagonal across samples) and takes u <- u + alpha ((u_hat - J^T lam+) - u)
 * with an l1-merit Armijo line search, until ||h||_inf < tol.  Everything is IEEE fp64.
 *
 * Conventions
 *   - Plain C, no torch types.  Every array argument named below "dev" is a DEVICE pointer owned by
 *     the caller (e.g. a torch tensor's data_ptr()); "host" pointers are host memory.  The library owns
 *     only the opaque problem handle and never allocates device memory in snap_project/snap_residual/
 *     snap_schur_apply (the caller supplies `workspace`); snap_project_host allocates a private
 *     staging area on first use and frees it in snap_problem_destroy.
 *   - Layout of a state (time-major, x fastest), dense, fp64:
 *         u[b][k][j][i]   b < batch, k < nt (time level), j < ny, i < nx      n = nt*ny*nx per sample
 *   - Layout of constraint rows / multipliers, per sample, m = snap_num_rows(p):
 *         local block [nt][ny][nx]: level 0 = initial-condition rows u[0] - u0 (Eq. 10, Eq. 14);
 *                                   level k >= 1 = one-step scheme residual between levels k-1 and k
 *                                   (PAPER.md L549, L561).  Kind HEAT1D_IC_MASS has level 0 only (nx rows).
 *         mass block  [nt]        : dx * sum_i u[k][i] - M0,  M0 = dx * sum_i u0[i],
 *                                   kinds HEAT1D_IC_MASS and BURGERS1D_LF_MASS only.
 *     Kind BURGERS1D_FLUXK, K = flux_steps, F = nt-1-K:  m = (K+1) nx + F + (energy_rows ? F : 0),
 *         local block [K+1][nx] (level 0 = IC rows, level k = residual of step k-1 -> k),
 *         mass block  [F]  levels K+1..nt-1 (the rows of levels 0..K are implied by the local rows and omitted,
 *                          as the paper omits its implied first row, L493),
 *         energy block [F] steps k = K..nt-2:  E(u[k+1]) - E(u[k]) + dt nu D(u[k]),  E(v) = dx/2 sum v_i^2,
 *                          D(v) = dx sum ((v_{i+1} - v_i)/dx)^2  (periodic), only if energy_rows != 0.
 *     (The paper lists IC, mass, flux rows in that order, L374/L499; row order only permutes lam.)
 *   - Asynchrony: device entry points only enqueue work on `stream` and return; per-sample outcome is in
 *     device memory (`iters`).  They never synchronise the host.
 *   - Errors: return value 0 = SNAP_OK, negative = error (see enum).  Non-convergence of an individual
 *     sample is NOT an error return: it is reported in iters[b] as a negative status.
 *   - Thread safety: distinct handles may be used concurrently; one handle must not be used from two
 *     host threads at once with the same workspace.
 */
#ifndef SNAP_H_
#define SNAP_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct snap_problem snap_problem; /* opaque, host side, owned by the library */
typedef void* snap_stream;                /* a cudaStream_t (NULL = legacy default stream) */

/* Constraint families (BASELINE.json configs 1..5). */
enum {
  SNAP_HEAT1D_IC_MASS = 0,    /* IC rows + per-level mass rows; affine (Eq. 10)                    */
  SNAP_BURGERS1D_LF = 1,      /* IC + finite-volume residual, Lax-Friedrichs flux, explicit viscosity, periodic  */
  SNAP_FISHER1D_IE = 2,       /* IC + implicit-Euler Fisher-KPP residual, ghost-cell Neumann                     */
  SNAP_ALLENCAHN2D_IE = 3,    /* IC + implicit-Euler Allen-Cahn residual, 5-point periodic (2D, PCG path)        */
  SNAP_BURGERS1D_LF_MASS = 4, /* kind 1 + per-level mass rows (dense border rows, all linearly dependent)        */
  SNAP_BURGERS1D_FLUXK = 5    /* the paper's "IC, Mass, Flux(k)" set (Eq. 14, Table XVIII): IC rows,
                                 finite-volume residual rows of the first flux_steps steps only (Lax-Friedrichs or
                                 Godunov flux, L555), a mass row per later level, optionally the energy-evolution row
                                 of Eq. 11 (L336, L603-607) per later step.  J is wide; the border rows are genuinely
                                 coupled (banded SPD Schur complement, banded Cholesky)       */
  ,
  SNAP_NS2D_VORT_ENST = 6     /* the paper's Navier-Stokes row set (Eq. 20): IC rows, total vorticity and enstrophy
                                 (dx dy sum w, dx dy sum w^2) of every later level.  No local PDE rows: the levels decouple
                                 and each is projected onto a sphere inside a hyperplane in closed form (2D, nx ny <= 4096,
                                 nt <= 2048).  m = ny nx + 2 (nt-1): [IC][vorticity nt-1][enstrophy nt-1]              */
};

/* Return codes. */
enum {
  SNAP_OK = 0,
  SNAP_EINVAL = -1,  /* bad kind / size / NULL pointer / ny != 1 for a 1D kind / size above the limits below */
  SNAP_ECUDA = -2,   /* a CUDA call or launch failed (query cudaGetLastError)                                */
  SNAP_ENOMEM = -3,  /* workspace too small / staging allocation failed                                       */
  SNAP_ELIMIT = -4   /* no-allocation entry point: batch*n exceeds the static scratch (SNAP_STATIC_SCRATCH_BYTES) */
};

/* Per-sample status written to iters[b] when negative; iters[b] >= 0 = number of linear (Schur) solves. */
enum {
  SNAP_ST_MAXITER = -1,    /* max_iter Gauss-Newton steps without reaching tol; u* = last iterate (kind
                              ALLENCAHN2D_IE: the last iterate of the INEXACT Newton sequence -- steps taken while
                              ||h||_inf >= tol are solved to the forcing tolerance of pcg_rtol below, so an
                              unconverged u* differs from an exactly solved sequence by that tolerance)           */
  SNAP_ST_LINESEARCH = -2, /* Armijo back-tracking exhausted ls_max halvings; u* = last accepted iterate      */
  SNAP_ST_NONFINITE = -3,  /* non-finite residual or direction; u* = u_hat, lam = 0          */
  SNAP_ST_PCG = -4         /* 2D: PCG hit pcg_max without reaching pcg_rtol; u* = last iterate               */
};

/* Which kernel served a sample (stats slot SNAP_STAT_VARIANT): a silent change of path is visible to callers. */
enum {
  SNAP_VAR_NONE = 0,
  SNAP_VAR_HEAT_CLOSED_FORM = 1, /* heat_project_kernel                                                          */
  SNAP_VAR_CLASSIC_BULK = 2,     /* project1d_kernel, rows by 1-D bulk (TMA) copies                               */
  SNAP_VAR_CLASSIC_PLAIN = 3,    /* project1d_kernel, plain loads/stores (odd nx / unaligned buffers)             */
  SNAP_VAR_FUSED_TMA = 4,        /* project1d_fused_kernel, tensor-map TMA rows, several GN iterations per pass   */
  SNAP_VAR_PCG2D = 5,            /* project2d_kernel: PCG on J J^T (precond 0, 1, 2)                              */
  SNAP_VAR_DIRECT2D = 6,         /* project2d_direct_kernel: product-form sweeps with in-SMEM level solves        */
  SNAP_VAR_FLUXK_BAND = 7,       /* project1d_fluxk_kernel: product form on the pinned levels + banded border solve */
  SNAP_VAR_NS_CLOSED_FORM = 8    /* ns_project_kernel: per-level sphere-in-hyperplane projection (kind 6)             */
};

/* Slots of one sample's work-counter record (snap_project_stats), 8 x int64. */
enum {
  SNAP_STAT_LINEARISATIONS = 0, /* Gauss-Newton linearisations (Schur solves, forward half) used               */
  SNAP_STAT_PASSES = 1,         /* passes over the time levels (forward, backward, correction sweeps)           */
  SNAP_STAT_ROWS_READ = 2,      /* HBM rows (one level of one field) requested for reading                      */
  SNAP_STAT_ROWS_WRITTEN = 3,   /* HBM rows written                                                             */
  SNAP_STAT_VARIANT = 4,        /* SNAP_VAR_*                                                                   */
  SNAP_STAT_INNER = 5,          /* 2D: PCG iterations (PCG path) / level-solve iterations (direct path)         */
  SNAP_STAT_ROW_DOUBLES = 6,    /* doubles per row: rows * row_doubles * 8 = algorithmic bytes                  */
  SNAP_STAT_BACKTRACKS = 7,     /* Armijo step-length reductions                                                */
  SNAP_STAT_COUNT = 8
};

/* Size limits of this implementation (snap_problem_create returns SNAP_EINVAL beyond them):
 *   1D kinds: 2 <= nx <= 512, ny == 1, 2 <= nt <= 65535;  2D kind: 4 <= nx, ny and nx*ny <= 4096, nt >= 2;
 *   kind BURGERS1D_FLUXK: nx in {32, 64, 128, 256}, nt <= 512 (the band system lives in shared memory). */

typedef struct {
  double dx, dy, dt;  /* grid steps (caller supplied so that oracle and GPU share them bit for bit)           */
  double nu, alpha;   /* Burgers: viscosity; Lax-Friedrichs dissipation (a constant)           */
  double D, rho;      /* Fisher-KPP: diffusion, reaction rate                                                 */
  double eps;         /* Allen-Cahn interface width                                                           */
  double tol;         /* stop when ||h(u)||_inf < tol                       (default 1e-10)                   */
  int max_iter;       /* cap on Gauss-Newton steps                          (default 50)                      */
  int polish;         /* extra full steps once tol is met; skipped when
                         ||h||_inf <= 1e-3 * tol already                    (default 1)                       */
  double ls_c1;       /* Armijo sufficient-decrease constant                (default 1e-4).  Kind HEAT1D_IC_MASS
                         has linear rows: the full Gauss-Newton step from u_hat IS the projection, the library
                         takes it in closed form and ls_c1 / ls_shrink / ls_max / max_iter are not consulted
                         (a merit test with ls_c1 >= 1/2 would reject that step: see DESIGN.md R25)               */
  double ls_shrink;   /* step-length reduction factor                       (default 0.5)                     */
  int ls_max;         /* maximum number of reductions per step              (default 20)                      */
  double pcg_rtol;    /* 2D: PCG stops at ||r - S lam||_2 <= pcg_rtol ||r||_2 (default 1e-13);
                         steps taken while ||h||_inf >= tol stop at ||r||_2 <= 1e-2 ||h||_inf ||h||_1/sqrt(n)
                         (never tighter than pcg_rtol ||b||, never looser than 1e-4 ||b||)                     */
  int pcg_max;        /* 2D: PCG iteration cap per solve                    (default 200)                     */
  int precond;        /* 2D: 0 none, 1 time-line, 2 time-line x ADI         (default 2)                       */
  int lambda_mode;    /* 0 = minimum-norm multiplier, 1 = basic (redundant multipliers = 0)    */
  int gn_fuse;        /* Burgers kinds (nx in {32,...,512}) and Fisher (nx in {32,...,256}): Gauss-Newton iterations carried by one
                         forward pass over the levels.  0 = as many as the kernel holds in
                         registers (default), k >= 1 = at most k, -1 = classic path (one forward and one
                         backward sweep per iteration).  Other kinds / sizes always take the classic path.   */
  int flux_steps;     /* kind BURGERS1D_FLUXK: K, number of leading steps that carry flux rows (0 <= K <= nt-1)     */
  int energy_rows;    /* kind BURGERS1D_FLUXK: 1 = add the energy-evolution row of every later step                  */
  int flux_kind;      /* kind BURGERS1D_FLUXK: 0 = Lax-Friedrichs (alpha), 1 = Godunov                               */
  int hessian;        /* 0 = Gauss-Newton, W = I (default, R1); 1 = exact Lagrangian Hessian
                         W = I + sum lam_i grad^2 h_i at the multipliers of the previous solve (Eq. 5,
                         Eq. 25), with an inertia safeguard per level (a level whose W_k has
                         an eigenvalue below 0.1 uses I).  It changes the step only where J is wide: kind BURGERS1D_FLUXK
                         with energy rows (quadratic instead of linear convergence); for the square kinds the step is
                         J du = -h whatever W is, and the setting is accepted and has no effect (R22).   */
} snap_params;

/* Fill *p with the defaults listed above (grid steps 1, physical constants 0, alpha = 1). */
void snap_params_default(snap_params* p);

/* Create a problem handle.  Validates kind/sizes/params, precomputes grid constants (and, for the 2D
 * kind, the truncated circulant Green's function of the ADI line operator, copied to device memory owned
 * by the handle).  ny must be 1 for 1D kinds.  *out is set only on success. */
int snap_problem_create(snap_problem** out, int kind, int nx, int ny, int nt, const snap_params* params);
int snap_problem_destroy(snap_problem* p);

/* Sizes: unknowns n and constraint rows m per sample (0 for a NULL handle). */
size_t snap_num_unknowns(const snap_problem* p);
size_t snap_num_rows(const snap_problem* p);

/* Bytes of device workspace snap_project needs for `batch` samples (any base alignment: the library aligns
 * inside the buffer and the figure includes the slack). */
size_t snap_workspace_bytes(const snap_problem* p, int batch);

/* Batched projection (Eq. 2/4; the whole hot path of SURVEY.md §8(a) a1-a9).
 *   u_hat   dev [batch][nt][ny][nx]  in   point to project.  May alias u_star (in place).
 *   cdata   dev [batch][ny][nx]      in   per-sample initial-condition target u0.
 *   u_star  dev [batch][nt][ny][nx]  out  projected field.
 *   lambda  dev [batch][m] or NULL   in/out  multipliers lam*.  NULL = multiplier-free call (PCFM's pull-back, PAPER.md
 *                                         Eq. 3, uses u* only): the product-form kernels then skip the y emission, the
 *                                         multiplier sweep and the min-norm correction (config 5: 40 n instead of 88 n
 *                                         bytes per projection); u*, status codes are unchanged, `iters` of the 2D
 *                                         product-form path is one short (the final multiplier linearisation is not run).
 *                                         Kernels that carry the multipliers in every iteration (classic sweeps, PCG, heat,
 *                                         kind 5) keep them in the tail of the workspace.
 *                                         If warm != 0 the incoming values are the PCG
 *                                         initial guess of the 2D kind; the 1D kinds solve
 *                                         directly and ignore them (R2/R3).  The iterate itself
 *                                         always starts at u_hat.
 *   iters   dev [batch] (int32)      out  number of Gauss-Newton linearisations (Schur solves, forward half)
 *                                         used, or a negative SNAP_ST_* status.
 *   workspace dev, workspace_bytes >= snap_workspace_bytes(p, batch); a shorter buffer returns SNAP_ENOMEM
 *             and nothing is launched.
 * Enqueues on `stream`; no host synchronisation. */
int snap_project(const snap_problem* p, int batch, const double* u_hat, const double* cdata, double* u_star,
                 double* lambda, int* iters, int warm, void* workspace, size_t workspace_bytes, snap_stream stream);

/* One PCFM sampling step around the projection (§III-A, Eq. 1-3), one launch
 * where the product-form kernels serve the problem (fused 1D path with one warp per sample, 2D product-form path):
 *     u_hat_1 = u_tau + (1 - tau) vel          Eq. 1, formed by the projection's first pass, written IN PLACE over u_tau
 *     u_1     = argmin 1/2 ||u - u_hat_1||^2 s.t. h(u) = 0     Eq. 2 = snap_project
 *     u_next  = u_prior + tau_next (u_1 - u_prior)             Eq. 3, written by the pass that streams the final iterate
 *   u_tau   dev [batch][n]  in: state at flow time tau; out: u_hat_1
 *   vel     dev [batch][n]  in: values of the flow model's velocity v_theta(u_tau, tau) (the model itself is the caller's)
 *   u_prior dev [batch][n]  in: the prior sample u_0 of the OT interpolant
 *   u1      dev [batch][n]  out: projected field;  u_next dev [batch][n] out;  the five field buffers must be distinct
 *   lambda  dev [batch][m] or NULL (multiplier-free step: what a sampler needs);  iters, workspace as snap_project.
 * Other kernels (classic sweeps, PCG, heat, kind 5) run Eq. 1 and Eq. 3 as two elementwise launches around theirs.
 * 0 <= tau, tau_next <= 1, else SNAP_EINVAL. */
int snap_flow_step(const snap_problem* p, int batch, double* u_tau, const double* vel, const double* u_prior, double tau,
                   double tau_next, const double* cdata, double* u1, double* u_next, double* lambda, int* iters,
                   void* workspace, size_t workspace_bytes, snap_stream stream);

/* Float32 mode (the paper's models are Float32 with solver tolerance 1e-5): the
 * multiplier-free projection of the Burgers kinds (BURGERS1D_LF, BURGERS1D_LF_MASS; nx in {32, 64, 128, 256}) computed
 * entirely in fp32 -- same method (forward passes carrying several Gauss-Newton iterations per level), full steps, stop
 * when ||h||_inf < tol (local and mass rows) and `polish` more steps were taken.  All field buffers are fp32, 16-byte aligned:
 *   u_hat dev [batch][nt][nx] in (may alias u_star), cdata dev [batch][nx] in, u_star dev [batch][nt][nx] out,
 *   iters dev [batch] out: residual evaluations used, or SNAP_ST_MAXITER / SNAP_ST_NONFINITE (u* = u_hat) /
 *   SNAP_ST_LINESEARCH (a full step that did not reduce ||h||_inf; u* = the iterate before it).
 *   tol > 0 (the paper's 1e-5); workspace as snap_project (only 2 n floats per sample are used).
 * Other kinds / sizes: SNAP_EINVAL. */
int snap_project_f32(const snap_problem* p, int batch, const float* u_hat, const float* cdata, float* u_star, int* iters,
                     float tol, void* workspace, size_t workspace_bytes, snap_stream stream);

/* Same computation with HOST buffers (pinned or pageable): copies inputs to a device staging area owned by
 * the handle, runs snap_project, copies u_star / lambda / iters back, and synchronises `stream` before
 * returning.  lambda is read only if warm != 0; lambda_host == NULL = multiplier-free call (no lambda copy either way). */
int snap_project_host(snap_problem* p, int batch, const double* u_hat_host, const double* cdata_host,
                      double* u_star_host, double* lambda_host, int* iters_host, int warm, snap_stream stream);

/* Constraint residual and the per-type norms of the paper's constraint-error metric
 * (Eq. 27).  Kind 6: the mass slot holds the total-vorticity rows, the energy slot the enstrophy rows.
 *   h      dev [batch][m] or NULL.
 *   norms  dev [batch][5] or NULL: ||h||_inf, ||h_IC||_2, ||h_PDE||_2, ||h_mass||_2, ||h_energy||_2 (0 where a type
 *          is absent). */
int snap_residual(const snap_problem* p, int batch, const double* u, const double* cdata, double* h,
                  double* norms, snap_stream stream);

/* Matrix-free Schur operator (SURVEY.md §8(a) a2+a4; kinds 0-4): out = J(u) J(u)^T x for x in the multiplier layout,
 * the operator is never assembled.  x, out: dev [batch][m]; u: dev [batch][nt][ny][nx].  `workspace` must
 * hold batch*n doubles (workspace_bytes >= batch*n*8, else SNAP_ENOMEM).  Used by the PCG path and exported for
 * validation against an assembled J J^T. */
int snap_schur_apply(const snap_problem* p, int batch, const double* u, const double* x, double* out,
                     void* workspace, size_t workspace_bytes, snap_stream stream);

/* No-allocation variant of snap_schur_apply, for callers that cannot allocate device memory or hand over a workspace
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The scratch vector
 * g = J(u)^T x lives in a file-scope `static __device__` array of SNAP_STATIC_SCRATCH_BYTES (8 MiB = 2^20 doubles) inside
 * the library; every GPU that loads libsnap holds those 8 MiB until the process exits.
 *   u, x, out   dev, as snap_schur_apply (kinds 0-4); same kernels, same result bit for bit.
 *   Limit       batch * n <= SNAP_STATIC_SCRATCH_BYTES / 8 = 1 048 576 (e.g. 64 samples of 128 x 128, 16 of 256 x 256);
 *               beyond it the call returns SNAP_ELIMIT and launches nothing.
 *   Allocation  the call performs no cudaMalloc / cudaFree and calls no allocating library routine; it enqueues two
 *               kernels on `stream` and returns.  The device address of the array is resolved once per device
 *               (cudaGetSymbolAddress, on the device current at that moment): by snap_static_scratch_init(), which a
 *               caller runs once per device at set-up (before stream capture), or else by the first call on that device.
 *   Sharing     there is ONE array per device, shared by every handle and every call, and it keeps the previous call's
 *               contents.  Nothing in it has to start at zero (each call overwrites every element it later reads), but two
 *               calls that overlap on the GPU (different streams, or graph branches without an edge between them) race
 *               on it: order them on one stream or with an event.  Use snap_schur_apply with private workspaces instead
 *               where calls must overlap.
 * snap_static_scratch_bytes() returns SNAP_STATIC_SCRATCH_BYTES. */
#define SNAP_STATIC_SCRATCH_BYTES 8388608
size_t snap_static_scratch_bytes(void);
int snap_static_scratch_init(void);
int snap_schur_apply_static(const snap_problem* p, int batch, const double* u, const double* x, double* out,
                            snap_stream stream);

/* Per-sample work counters of the most recent snap_project call that used `workspace` with the same `batch`,
 * copied on `stream` into
 *   stats  dev [batch][SNAP_STAT_COUNT] (int64), slots SNAP_STAT_* above.
 * (rows read + rows written) * row_doubles * 8 is the traffic the method itself asked for (bench.py's
 * algorithmic bytes); the variant slot says which kernel ran. */
int snap_project_stats(const snap_problem* p, int batch, const void* workspace, size_t workspace_bytes,
                       long long* stats, snap_stream stream);

/* Number of kernel launches the library has enqueued through this handle since creation (host counter). */
long long snap_launch_count(const snap_problem* p);

const char* snap_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* SNAP_H_ */
