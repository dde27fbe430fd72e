/*
 * mhs.h -- C ABI of libmhs_b200: the B200 (sm_100a) multigrid solve for the poloidal scalar
 * potential P of linear magnetohydrostatic equilibria, after MacTaggart, Elsheikh, McLaughlin &
 * Simitev, "Non-symmetric magnetohydrostatic equilibria: a multigrid approach" (arXiv 1307.6720).
 * Citations "PAPER.md:<line>" refer to the paper text; "C<n>" to the readings listed in DESIGN.md.
 *
 * The library follows the paper's procedure (restated :224-247):
 *     1. P = 0 everywhere
 *     2. 2D multigrid for  P_xx + P_yy = -B_z(x,y)  on z = 0, P = 0 on the edges   (eq 11, :94, :99)
 *     3. 3D multigrid for  (1+f(z)) (P_xx + P_yy) + P_zz + alpha^2 P = 0     (eq 8, :67, :100)
 *        with P = 0 on the side and top boundaries and step 2's P on the bottom;  f = -xi (C1)
 *     4. B, p, rho by second-order central finite differences               (:102-113, eqs 9, 10)
 * Multigrid = V(n_pre,n_post) cycles of weighted Gauss-Jacobi relaxation, residual, full-weighting
 * "reduction" and tri/bi-linear prolongation (the four components of PAPER.md:210), rediscretised
 * coarse operators, exact solve on the coarsest level, stop on ||r_k||_2 <= tol ||r_0||_2 (C4-C10).
 *
 * Conventions
 *   Grid      vertex grid nx x ny x nz INCLUDING boundary nodes on [0,Lx]x[0,Ly]x[0,Lz]; every
 *             extent must be 2^m q + 1 with m >= 1 (>= 3 nodes).  (C2)
 *   Layout    every array crossing this ABI is DENSE, x fastest: idx = i + nx*(j + ny*k)
 *             (PAPER.md:214-216), element type float or double as chosen by mhs_options.dtype.
 *   Memory    "device" pointers are CUDA device pointers on the current device, "host" pointers
 *             are ordinary host memory (pinned for best speed).  The caller owns every buffer it
 *             passes; the library copies what it keeps (f_profile, p_b, rho_b, dfdz) and owns the
 *             context and its internal hierarchy, all allocated in mhs_create -- the device-pointer
 *             calls (mhs_solve_*, mhs_fields, ...) allocate nothing on the device.  The *_host entry
 *             points are the exception: the first mhs_fields_host* / mhs_get_potential_host call
 *             allocates a device staging buffer (5N resp. N elements, kept until mhs_destroy), and
 *             event timing (mhs_options.profile > 0) creates CUDA events on demand and recycles them.
 *   Streams   all work is enqueued on mhs_options.stream (a cudaStream_t; NULL = default stream).
 *             mhs_solve_* return after the last residual norm has been read back (they report
 *             `cycles`); the other calls are asynchronous with respect to the host unless they
 *             take a host pointer, in which case they return after the copy has completed.
 *   Errors    status codes only; nothing throws or aborts across the ABI.  On any error other
 *             than MHS_ERR_NOT_CONVERGED outputs are unspecified/untouched; mhs_last_error()
 *             gives a message.  There is no CPU fallback: without a usable CUDA device
 *             mhs_create fails with MHS_ERR_CUDA.
 *   State     create -> solve_boundary -> solve_interior (repeatable: it CONTINUES from the
 *             current P, so max_cycles = 1 called k times yields iterate k) -> fields.
 *             solve_boundary resets the interior to 0.  mhs_solve_interior and
 *             mhs_fields* before a successful mhs_solve_boundary (MHS_OK or MHS_ERR_NOT_CONVERGED)
 *             or mhs_set_potential return MHS_ERR_STATE.
 */
#ifndef MHS_H_
#define MHS_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mhs_ctx mhs_ctx; /* opaque, library-owned; one per grid + stream; not thread-safe */

typedef enum {
    MHS_OK = 0,
    MHS_ERR_INVALID_ARG = 1,
    MHS_ERR_GRID = 2,          /* an extent is not 2^m*q+1 with m>=1, or the coarsest level is too large */
    MHS_ERR_NOT_ELLIPTIC = 3,  /* some 1 + f(z_k) <= 0, i.e. xi >= 1       */
    MHS_ERR_INDEFINITE = 4,    /* some diagonal D_k >= 0 on some level (alpha^2 too large for the grid) */
    MHS_ERR_STATE = 5,         /* call order violated                                                  */
    MHS_ERR_NOT_CONVERGED = 6, /* max_cycles reached; the result is still the valid k-th iterate       */
    MHS_ERR_CUDA = 7,
    MHS_ERR_OOM = 8
} mhs_status;

typedef struct { int nx, ny, nz; double Lx, Ly, Lz; } mhs_grid;

#define MHS_BC_DIRICHLET_ZERO 0 /* P = 0 on the face: the paper's choice                                     */
#define MHS_BC_DIRICHLET_DATA 1 /* P given on the face by mhs_set_wall_data ("In principle other elliptic
                                   equations can be defined on the other boundaries")                  */
typedef struct { int sides, top; } mhs_bc; /* the four side faces / the top face; NULL = both MHS_BC_DIRICHLET_ZERO */

#define MHS_F32 0
#define MHS_F64 1

/* mhs_options.flags */
#define MHS_FLAG_REFERENCE_KERNELS 1 /* one thread per node, one kernel per operator, no fusion: the
                                        paper's own kernel design; for A/B tests */
#define MHS_FLAG_UNFUSED_KERNELS    4 /* tuned kernels, but one sweep per pass (no temporal blocking);
                                        for A/B tests of the fused smoother                              */
#define MHS_FLAG_BIG_LEVEL_KERNELS  8 /* use the kernels of the big (HBM-bound) levels on every level they
                                        can handle, whatever its size; for parity tests on small grids     */
#define MHS_FLAG_SEPARATE_PROLONG  16 /* keep the prolongation a pass of its own instead of folding it into the
                                        first post-smoothing pass of the big levels; for A/B tests              */
#define MHS_FLAG_NO_PDL            32 /* launch every kernel fully serialised (no programmatic dependent launch)   */
#define MHS_FLAG_LOADED_RESTRICT   64 /* finest level: residual + restriction by the kernel that loads through the L1
                                        instead of the bulk-copy fed one; for A/B tests                         */
#define MHS_FLAG_LOADED_FIELDS    128 /* mhs_fields by the register z-streaming kernel instead of the bulk-copy fed
                                        one; for A/B tests                                                      */
#define MHS_FLAG_NO_FOLDED_NORM   256 /* keep the stop rule a kernel launch of its own instead of folding it into the finest
                                        level's restriction kernel; for A/B tests                                    */
#define MHS_FLAG_SYNC_EACH_CYCLE   2 /* read the norm back after every cycle instead of running
                                        cycles speculatively behind a device-side stop flag          */

/* mhs_options.smoother (reading C25) */
#define MHS_SMOOTH_JACOBI 0 /* weighted point Gauss-Jacobi: the paper's relaxation             */
#define MHS_SMOOTH_ZLINE  1 /* weighted z-line Jacobi, u' = u + omega T^-1 (rhs - L u), T = diagonal of L + its two
                               z-neighbours, one tridiagonal solve per (i,j) line: for strong (1 - xi) anisotropy --
                               the paper's xi_2 profile reaches 1 - xi = 0.05.  3D solve only; the 2D
                               boundary solve keeps point Jacobi.  Every level runs general one-pass kernels (no
                               temporal blocking, no shared-memory tail).                                          */

typedef struct {
    int dtype;                 /* MHS_F32 / MHS_F64: element type of ALL device/host field arrays      */
    double omega;              /* Jacobi weight (C4); benchmarks use 2/3                               */
    int n_pre, n_post;         /* sweeps before / after the coarse-grid correction (C5)                */
    int max_levels;            /* 0 = coarsen fully (C8)                                               */
    double boundary_tol;       /* relative tolerance of the 2D solve (C11)                             */
    int boundary_max_cycles;
    double mu0, g;             /* eqs (9), (10)                                                        */
    const double *p_b, *rho_b; /* host, nz each; NULL -> zeros                                         */
    const double *dfdz;        /* host, nz; NULL -> finite differences of f_profile (C14)              */
    void *stream;              /* cudaStream_t                                                         */
    int profile;               /* 1: time every kernel class with CUDA events on `stream`              */
    int flags;                 /* MHS_FLAG_*                                                           */
    int smoother;              /* MHS_SMOOTH_JACOBI (default) / MHS_SMOOTH_ZLINE                       */
    int fmg_cycles;            /* 0 (default): the interior starts from P = 0 as the paper's step 1 says.
                                  n > 0: FULL-MULTIGRID START (reading C26) -- the first mhs_solve_interior after
                                  mhs_solve_boundary (not after mhs_set_potential: a potential the caller gives is
                                  continued from) first replaces the interior by a guess built
                                  from the coarse grids upwards: level l carries the bottom data by injection, the
                                  coarsest level is solved exactly, every finer level starts from the trilinear
                                  interpolation of the level below and gets n V-cycles; the ordinary cycles follow.
                                  r0 stays the residual norm of the zero-interior iterate, so `tol` means the same;
                                  info.cycles counts the ordinary finest-level cycles only (0 if the FMG iterate
                                  already meets the tolerance).                                          */
} mhs_options;

#define MHS_HISTORY_LEN 256
typedef struct {
    int cycles;                       /* V-cycles performed by this call                               */
    double r0;                        /* ||rhs - L u||_2 of the initial iterate (zero interior)        */
    double r_final;                   /* after the last cycle                                          */
    double history[MHS_HISTORY_LEN];  /* history[k] = norm after cycle k+1 of this call                */
    int stagnated;                    /* fp32 only (C20): stopped because r_k > 0.9 r_{k-1} twice in a
                                         row -- the fp32 residual floor; reported as MHS_OK          */
} mhs_solve_info;

/* Kernel classes for mhs_profile. */
enum {
    MHS_KC_SMOOTH_L0 = 0,   /* Jacobi sweeps on the finest 3D level (the dominant, HBM-bound kernel) */
    MHS_KC_RESTRICT_L0 = 1, /* residual + full weighting on the finest 3D level                      */
    MHS_KC_PROLONG_L0 = 2,  /* trilinear correction on the finest 3D level (alone, or fused with the
                               first post-smoothing pass: see mhs_profile.fused_prolong_l0)          */
    MHS_KC_NORM_L0 = 3,     /* residual norm on the finest 3D level                                  */
    MHS_KC_COARSE_3D = 4,   /* everything on 3D levels >= 1                                          */
    MHS_KC_BOUNDARY_2D = 5, /* the whole 2D solve                                                    */
    MHS_KC_FIELDS = 6,      /* B, p, rho                                                             */
    MHS_KC_PACK = 7,        /* dense <-> internal layout, zero fills                                 */
    MHS_KC_COUNT = 8
};
typedef struct {
    long long launches[MHS_KC_COUNT]; /* kernels launched per class since create / reset             */
    double ms[MHS_KC_COUNT];          /* CUDA-event time per class (options.profile = 1: the smoothing and
                                         prolongation classes of the finest level only; 2: every class)  */
    long long sweeps_l0;              /* Jacobi sweeps applied to the finest 3D level                */
    long long fused_prolong_l0;       /* launches of class MHS_KC_PROLONG_L0 that were prolongation-fused
                                         smoothing passes (prolongation + the first post-sweeps in one pass) */
    long long xtiled_zsweep;          /* launches of the temporally blocked smoother (any level) whose tiles were
                                         narrower than a grid row (rows wider than 256 fp64 / 512 fp32 columns)  */
    long long ring_restrict;          /* residual + restriction launches (any level) that ran in the bulk-copy fed
                                         kernel                                                                 */
    long long ring_fields;            /* mhs_fields calls served by the bulk-copy fed kernel                    */
} mhs_profile;

/* Fill *o with the defaults: fp64, omega 2/3, V(2,2), full coarsening, boundary_tol 1e-10,
 * boundary_max_cycles 100, mu0 = 1/2, g = 1 (C16), no profiles, default stream, point Jacobi, no FMG start. */
void mhs_default_options(mhs_options *o);

/* Build a context: level hierarchy (C8), per-level coefficient tables c_l[k] = 1 + f(z_k) injected
 * to the coarse levels (C7), omega/D_k, inverse of the coarsest operators (C9), device arrays.
 * f_profile: host, nz doubles, f(z_k) at the nodes (NULL -> 0: the force-free case).
 * bc: NULL or all MHS_BC_DIRICHLET_ZERO.  opts: NULL -> defaults.  P is initialised to 0 (step 1).
 * grid->nz == 1 makes a BOUNDARY-ONLY context: only eq (11) on the nx x ny plane is set up (step 2 of the
 * procedure); mhs_solve_boundary works and its result is read with mhs_level_get(ctx, 2, 0, 0, P0),
 * the interior / field calls return MHS_ERR_STATE. */
mhs_status mhs_create(const mhs_grid *grid, double alpha, const double *f_profile, const mhs_bc *bc,
                      const mhs_options *opts, mhs_ctx **out);
void mhs_destroy(mhs_ctx *ctx);

/* Steps 1-2 (eq 11): P = 0 everywhere, then 2D V-cycles for L2 P0 = -Bz0 with
 * P0 = 0 on the edges until ||r|| <= boundary_tol ||r0|| or boundary_max_cycles; P(:,:,0) = P0.
 * Bz0: nx*ny values (dtype), device / host.  info may be NULL. */
mhs_status mhs_solve_boundary(mhs_ctx *ctx, const void *Bz0_device, mhs_solve_info *info);
mhs_status mhs_solve_boundary_host(mhs_ctx *ctx, const void *Bz0_host, mhs_solve_info *info);

/* Step 3 (eq 8): V-cycles on the interior, continuing from the current P, until
 * ||r_k|| <= tol * r0 or max_cycles cycles have been done in this call (1 <= max_cycles).
 * r0 is the residual norm of the iterate found at the first call after mhs_solve_boundary /
 * mhs_set_potential and is remembered across continuing calls. */
mhs_status mhs_solve_interior(mhs_ctx *ctx, double tol, int max_cycles, mhs_solve_info *info);

/* A batch of nb magnetograms on ONE context -- e.g. a time series of the same region feeding an MHD code (
 * SURVEY 8(f) NEXT-3): for b = 0 .. nb-1 in order the paper's whole procedure, mhs_solve_boundary(Bz0 + b nx ny) ->
 * mhs_solve_interior(tol, max_cycles) -> whichever outputs are non-NULL, member b at offset b times the member's size:
 * P (N values per member), B (3N), p (N), rho (N).  All device, dense, the context's dtype.  infos: host array of nb
 * mhs_solve_info of the interior solves, or NULL.  Member by member the results are those of the separate calls (each
 * member starts from P = 0).  Returns MHS_OK; MHS_ERR_NOT_CONVERGED if some member reached max_cycles (every
 * member is still computed and stored); otherwise the first error, with the members before it complete. */
mhs_status mhs_solve_batch(mhs_ctx *ctx, int nb, const void *Bz0_device, double tol, int max_cycles, void *P_device,
                           void *B_device, void *p_device, void *rho_device, mhs_solve_info *infos);

/* Field recovery (C13-C15).  B: 3*N values, Bx | By | Bz one after the other;
 * p, rho: N values each, N = nx*ny*nz.  Any of B, p, rho may be NULL (skipped). */
mhs_status mhs_fields(mhs_ctx *ctx, void *B_device, void *p_device, void *rho_device);
mhs_status mhs_fields_host(mhs_ctx *ctx, void *B_host, void *p_host, void *rho_host);
/* Diagnostics of the recovered field (the quantities of the paper's Figs 2, 4-7): |B| and the current
 * density j = curl B / mu0 (eq 2) with |j|, by second-order central differences of B (one-sided second order
 * in z on the bottom plane; j = 0 on the side and top boundary nodes, where B = 0 is imposed).
 * B_device: the 3*N values mhs_fields wrote (Bx | By | Bz).  absB, absJ: N values; J: 3*N (jx | jy | jz); any of the three
 * outputs may be NULL (skipped).  All device, dense, the context's dtype. */
mhs_status mhs_diagnostics(mhs_ctx *ctx, const void *B_device, void *absB_device, void *J_device, void *absJ_device);
/* Field-line integration (the field lines of the paper's Figs 1, 4, 5; reading C24): for every
 * seed the line  dx/ds = direction * B(x) / |B(x)|  (s = arc length) is followed with the classical fourth-order Runge-Kutta
 * method and a fixed step `step`; B between the nodes is the trilinear interpolation of the nodal B (cell = floor(x/hx) clamped
 * to the grid, lerp along x, then y, then z).  Point 0 of a line is its seed; the line ends when a Runge-Kutta stage or the new
 * point lies outside [0,Lx]x[0,Ly]x[0,Lz], when |B| <= bmin at a stage (a null point), or at max_points points.
 * A seed outside the box gives 0 points.  Nothing is rendered: the polylines are left in a device buffer.
 *   B_device     3*N values as mhs_fields wrote them (Bx | By | Bz), dense, the context's dtype
 *   seeds_device 3*nseeds values (x, y, z per seed), the context's dtype, coordinates in [0,Lx]x[0,Ly]x[0,Lz]
 *   lines_device nseeds * max_points * 3 values: point n of line s at [(s*max_points + n)*3 + {0,1,2}]; entries beyond a
 *                line's point count are left untouched
 *   npoints_device nseeds ints: points written per line
 * direction: +1 along B, -1 against it.  step > 0, max_points >= 1, bmin >= 0.  Asynchronous on the context's stream.
 * In fp64 every product-sum is one fma, in the order: lerps fma(t, b - a, a); |B|^2 = fma(bz,bz, fma(by,by, bx*bx));
 * stage points fma(step/2 or step, k, x); new point fma(step/6, (k1 + k4) + 2 (k2 + k3), x). */
mhs_status mhs_fieldlines(mhs_ctx *ctx, const void *B_device, int nseeds, const void *seeds_device, double step, int max_points,
                          int direction, double bmin, void *lines_device, int *npoints_device);
/* The same without waiting for the copies: the fields are computed on the context's stream into the library's staging
 * buffer and copied to the (pinned) host buffers on a separate copy stream; the call returns as soon as that is enqueued,
 * so the next mhs_solve_* can run while the results of this one travel over PCIe.  The host buffers must not be read, and
 * must stay valid, until mhs_host_sync() has returned.  A later mhs_fields_host* / mhs_get_potential_host first waits
 * (on the device) for the pending copies, so one staging buffer serves any pipeline depth. */
mhs_status mhs_fields_host_async(mhs_ctx *ctx, void *B_host, void *p_host, void *rho_host);
/* Block until every copy enqueued by mhs_fields_host_async has landed in host memory. */
mhs_status mhs_host_sync(mhs_ctx *ctx);

/* Read / overwrite the current iterate P (N values, dense).  mhs_set_potential takes the interior
 * and bottom-plane interior values; side/top/bottom-edge values of the input are ignored (they
 * are the Dirichlet zeros).  Needed for per-iterate parity checks and for resuming a solve. */
mhs_status mhs_get_potential(mhs_ctx *ctx, void *P_device);
mhs_status mhs_get_potential_host(mhs_ctx *ctx, void *P_host);
mhs_status mhs_set_potential(mhs_ctx *ctx, const void *P_device);

/* The result of the last mhs_solve_boundary alone: P(x,y,0), nx*ny values, dense (step 2).  Works on a
 * boundary-only context (nz = 1) too.  The host variant returns after the copy has completed. */
mhs_status mhs_get_boundary(mhs_ctx *ctx, void *P0_device);
mhs_status mhs_get_boundary_host(mhs_ctx *ctx, void *P0_host);

const char *mhs_last_error(const mhs_ctx *ctx); /* never NULL; valid until the next call on ctx */
const char *mhs_status_string(mhs_status s);

/* ---- instrumentation ------------------------------------------------------------------------ */
mhs_status mhs_get_profile(mhs_ctx *ctx, mhs_profile *out); /* synchronises the stream             */
/* Change mhs_options.profile (0: launch counts only; 1: CUDA events around the finest-level smoothing / prolongation
 * launches; 2: around every kernel class).  Event records between kernels undo the overlap of dependent launches and of
 * the copy stream, so timing runs that are not about kernel shares should use 0. */
mhs_status mhs_set_profiling(mhs_ctx *ctx, int level);
mhs_status mhs_reset_profile(mhs_ctx *ctx);
const char *mhs_kernel_class_name(int kernel_class);

/* ---- operator-level access (tests and micro-benchmarks of single multigrid components) -------
 * dim = 2 (boundary hierarchy) or 3 (interior hierarchy); level 0 is the finest.
 * which: 0 = u (the iterate / correction), 1 = rhs, 2 = r (residual scratch).  The finest 3D level
 * has rhs == 0 and no rhs array (MHS_ERR_INVALID_ARG).  Arrays are dense, that level's extents. */
int mhs_num_levels(const mhs_ctx *ctx, int dim);
mhs_status mhs_level_dims(const mhs_ctx *ctx, int dim, int level, int *nx, int *ny, int *nz);
mhs_status mhs_level_set(mhs_ctx *ctx, int dim, int level, int which, const void *src_device);
mhs_status mhs_level_get(mhs_ctx *ctx, int dim, int level, int which, void *dst_device);
mhs_status mhs_op_smooth(mhs_ctx *ctx, int dim, int level, int sweeps);   /* u <- S^sweeps u          */
mhs_status mhs_op_residual(mhs_ctx *ctx, int dim, int level);             /* r <- rhs - L u           */
mhs_status mhs_op_restrict(mhs_ctx *ctx, int dim, int level);             /* rhs_{l+1} <- R (rhs - L u)_l */
mhs_status mhs_op_prolong(mhs_ctx *ctx, int dim, int level);              /* u_l <- u_l + P u_{l+1}   */
mhs_status mhs_op_vcycle(mhs_ctx *ctx, int dim, int level);               /* one V-cycle from `level`: level 0
                                                                             continues from u, levels >= 1 start
                                                                             from u = 0 as inside a cycle      */
mhs_status mhs_op_resnorm(mhs_ctx *ctx, int dim, int level, double *out_host); /* ||rhs - L u||_2     */

/* Dirichlet data for P on the side and top faces (contexts created with MHS_BC_DIRICHLET_DATA in mhs_bc.sides and / or
 * .top; MHS_ERR_STATE otherwise).  G_device: a DENSE nx*ny*nz array of the context's dtype (device) of which only the nodes on
 * faces declared MHS_BC_DIRICHLET_DATA are read -- side nodes i = 0, nx-1 or j = 0, ny-1 on every plane k (the rim of the
 * bottom plane included), top nodes k = nz-1 away from the rim; faces declared MHS_BC_DIRICHLET_ZERO keep P = 0.  The values
 * would come from whatever problems are posed on those faces (a boundary-only context, nz = 1, solves eq 11 on a face).
 * The data is copied; it stays in force until the next call (mhs_solve_boundary resets the interior, not the walls).  Until
 * the first call the walls are zero.  Such a context solves  eq 8  with P = G on those faces: internally P = P_h + W, W = the
 * wall values, P_h with zero walls and the right-hand side -L W on the finest level (it allocates that array, W and one dense
 * scratch array in mhs_create: 3N elements more); mhs_get_potential and mhs_fields return the full P and its fields
 * (B = 0 on side and top nodes as before, C13; the nodes next to them take the wall values through the central differences),
 * the latter by the general one-thread-per-node kernel.  mhs_set_potential sets P_h: the wall nodes of its argument are
 * ignored.  Needs the point-Jacobi smoother and fmg_cycles = 0 (mhs_create: MHS_ERR_INVALID_ARG otherwise).               */
mhs_status mhs_set_wall_data(mhs_ctx *ctx, const void *G_device);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the residual norm of eq 8 (the quantity of the stop rule, C10),
 *     *out_device = || [c_k (D_xx + D_yy) + D_zz + alpha^2] P ||_2   over the interior nodes,  c_k = 1 + f(z_k) = 1 - xi(z_k),
 * of a DENSE potential P (nx*ny*nz elements of `dtype`, device; boundary nodes included and read as they are).  It
 * needs no mhs_ctx and calls no cudaMalloc / cudaFree or allocating library routine: its partial sums live in a
 * file-scope device array of MHS_STATIC_SCRATCH_DOUBLES doubles (512 KB, held by every GPU that loads the library
 * until the process exits).  One partial sum per 8 rows of a plane: grids with ceil((ny-2)/8) * (nz-2) >
 * MHS_STATIC_SCRATCH_DOUBLES (or nz - 2 > 65535) are rejected with MHS_ERR_INVALID_ARG (513^3 needs 32704, 1025 x 1025 x 257
 * 32640).  c_device: nz doubles on the device.  hx, hy, hz: mesh widths.  stream: a cudaStream_t (NULL = default
 * stream); the call is asynchronous, the result is ordered on `stream`.  Every call shares the one scratch array:
 * calls that overlap on the GPU race.  The array keeps the last call's contents; no call depends on them.
 * mhs_static_last_error(): message of the calling thread's last failed mhs_resnorm_static.                          */
#define MHS_STATIC_SCRATCH_DOUBLES 65536
mhs_status mhs_resnorm_static(const void *P_device, int dtype, int nx, int ny, int nz, double hx, double hy, double hz,
                              double alpha, const double *c_device, double *out_device, void *stream);
const char *mhs_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MHS_H_ */
