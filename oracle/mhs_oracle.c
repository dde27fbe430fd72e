/*
 * oracle/mhs_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU (fp64, scalar triple loops, one array per
 * quantity, no fusion, no blocking) implementation of the hot path of
 * MacTaggart, Elsheikh, McLaughlin & Simitev, "Non-symmetric magnetohydrostatic
 * equilibria: a multigrid approach" (arXiv 1307.6720; /root/reference/PAPER.md):
 *
 *   step 1  P = 0 everywhere
 *   step 2  2D multigrid for  P_xx + P_yy = -B_z  on z = 0       PAPER.md:94 (eq 11), :99
 *   step 3  3D multigrid for  [1-xi(z)](P_xx+P_yy)+P_zz+a^2 P=0  PAPER.md:67 (eq 8),  :100
 *   then    B, p, rho by 2nd-order central finite differences    PAPER.md:102-113, eqs 9,10
 *
 * The multigrid components are the four the paper lists: Gauss-Jacobi
 * relaxation (two arrays, separate boundary branch: PAPER.md:218), residual, "reduction"
 * (restriction) and prolongation.  Where the paper is silent the readings are those of
 * SURVEY.md section 8(c) / DESIGN.md "Readings" (C1..C23): weighted Jacobi (omega option),
 * V(nu1,nu2), full weighting, tri/bi-linear interpolation, rediscretised coarse operators
 * with injected coefficient, exact dense solve on the coarsest level, unweighted l2 norm
 * of rhs - L u over interior nodes.  xi(z) = -f(z)  (C1), so the operator is
 * (1+f(z))(P_xx+P_yy) + P_zz + alpha^2 P.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path.
 * Every function has a pin in tests/test_oracle_pins.py, orc_diagnostics in tests/test_diagnostics.py (see DESIGN.md
 * "Oracle and its pins");
 * values printed by the paper for P, B, p, rho do not exist (PAPER.md has none), so
 * "paper-value parity" is unpinned and closed forms / invariants / brute force replace it.
 *
 * Arrays are dense, x fastest: idx = i + nx*(j + ny*k).
 * OpenMP pragmas (only when compiled with -fopenmp) sit on loops whose iterations are
 * independent, so results are bit-identical with any thread count; norms stay serial.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define I3(i, j, k) ((size_t)(i) + (size_t)nx * ((size_t)(j) + (size_t)ny * (size_t)(k)))
#define I2(i, j) ((size_t)(i) + (size_t)nx * (size_t)(j))

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * Level rule (SURVEY 8(c) "create", reading C8): level l (0 = finest) is the coarsest when
 * any axis has an odd number of intervals or fewer than 4 intervals, or l+1 == max_levels
 * (max_levels = 0: coarsen fully).  nz <= 1 means "2D" and the z axis is ignored.
 * ---------------------------------------------------------------------------------- */
int orc_is_coarsest(int nx, int ny, int nz, int level, int max_levels)
{
    int mx = nx - 1, my = ny - 1, mz = nz - 1;
    if (max_levels > 0 && level + 1 >= max_levels) return 1;
    if ((mx % 2) || mx < 4) return 1;
    if ((my % 2) || my < 4) return 1;
    if (nz > 1 && ((mz % 2) || mz < 4)) return 1;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Dense Gaussian elimination with partial pivoting, A (n x n, row major) and b are
 * overwritten, solution returned in b.  Returns 0, or -1 on a zero pivot.  (C9)
 * ---------------------------------------------------------------------------------- */
int orc_dense_solve(int n, double *A, double *b)
{
    for (int col = 0; col < n; ++col) {
        int piv = col;
        double best = fabs(A[(size_t)col * n + col]);
        for (int r = col + 1; r < n; ++r) {
            double v = fabs(A[(size_t)r * n + col]);
            if (v > best) { best = v; piv = r; }
        }
        if (best == 0.0) return -1;
        if (piv != col) {
            for (int c = 0; c < n; ++c) {
                double t = A[(size_t)col * n + c];
                A[(size_t)col * n + c] = A[(size_t)piv * n + c];
                A[(size_t)piv * n + c] = t;
            }
            double t = b[col]; b[col] = b[piv]; b[piv] = t;
        }
        for (int r = col + 1; r < n; ++r) {
            double m = A[(size_t)r * n + col] / A[(size_t)col * n + col];
            if (m == 0.0) continue;
            for (int c = col; c < n; ++c) A[(size_t)r * n + c] -= m * A[(size_t)col * n + c];
            b[r] -= m * b[col];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        double s = b[r];
        for (int c = r + 1; c < n; ++c) s -= A[(size_t)r * n + c] * b[c];
        b[r] = s / A[(size_t)r * n + r];
    }
    return 0;
}

/* ====================================================================================
 *                                       3D
 *  (L u)_ijk = c_k [ (u_{i+1}-2u+u_{i-1})/hx^2 + (u_{j+1}-2u+u_{j-1})/hy^2 ]
 *              + (u_{k+1}-2u+u_{k-1})/hz^2 + alpha^2 u,   c_k = 1 + f(z_k) = 1 - xi(z_k)
 *  second-order central differences of eq (8)
 * ================================================================================== */

/* out = L u at interior nodes, 0 on boundary nodes. */
void orc_apply3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                double alpha, const double *u, double *out)
{
    memset(out, 0, sizeof(double) * (size_t)nx * ny * nz);
#pragma omp parallel for schedule(static)
    for (int k = 1; k < nz - 1; ++k)
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                double uc = u[I3(i, j, k)];
                double dxx = (u[I3(i + 1, j, k)] - 2.0 * uc + u[I3(i - 1, j, k)]) / (hx * hx);
                double dyy = (u[I3(i, j + 1, k)] - 2.0 * uc + u[I3(i, j - 1, k)]) / (hy * hy);
                double dzz = (u[I3(i, j, k + 1)] - 2.0 * uc + u[I3(i, j, k - 1)]) / (hz * hz);
                out[I3(i, j, k)] = c[k] * (dxx + dyy) + dzz + alpha * alpha * uc;
            }
}

/* Diagonal of L on plane k (D_k). */
static double diag3(double hx, double hy, double hz, double ck, double alpha)
{
    return -2.0 * ck / (hx * hx) - 2.0 * ck / (hy * hy) - 2.0 / (hz * hz) + alpha * alpha;
}

/* r = rhs - L u at interior nodes, 0 on boundary ("calculation of the residual").
 * rhs may be NULL (== 0). */
void orc_residual3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                   double alpha, const double *u, const double *rhs, double *r)
{
    orc_apply3(nx, ny, nz, hx, hy, hz, c, alpha, u, r);
#pragma omp parallel for schedule(static)
    for (int k = 1; k < nz - 1; ++k)
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                size_t p = I3(i, j, k);
                r[p] = (rhs ? rhs[p] : 0.0) - r[p];
            }
}

/* One weighted Gauss-Jacobi sweep, two arrays (old values read from one array,
 * new values written to the other; "one command for points on the boundary and another for
 * points in the interior"):  boundary: unew = u;  interior: unew = u + (omega/D_k)(rhs - L u). */
void orc_jacobi3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                 double alpha, double omega, const double *u, const double *rhs, double *unew)
{
    memcpy(unew, u, sizeof(double) * (size_t)nx * ny * nz); /* boundary branch */
#pragma omp parallel for schedule(static)
    for (int k = 1; k < nz - 1; ++k) {
        double D = diag3(hx, hy, hz, c[k], alpha);
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                size_t p = I3(i, j, k);
                double uc = u[p];
                double dxx = (u[I3(i + 1, j, k)] - 2.0 * uc + u[I3(i - 1, j, k)]) / (hx * hx);
                double dyy = (u[I3(i, j + 1, k)] - 2.0 * uc + u[I3(i, j - 1, k)]) / (hy * hy);
                double dzz = (u[I3(i, j, k + 1)] - 2.0 * uc + u[I3(i, j, k - 1)]) / (hz * hz);
                double Lu = c[k] * (dxx + dyy) + dzz + alpha * alpha * uc;
                unew[p] = uc + (omega / D) * ((rhs ? rhs[p] : 0.0) - Lu);
            }
    }
}

/* Full-weighting restriction ("reduction"; reading C6):
 * rc[I,J,K] = sum_{a,b,c in {-1,0,1}} w_a w_b w_c r[2I+a,2J+b,2K+c], w = (1/4,1/2,1/4),
 * at coarse interior nodes; 0 on the coarse boundary.  (nx,ny,nz) is the FINE grid. */
void orc_restrict3(int nx, int ny, int nz, const double *r, double *rc)
{
    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1, cz = (nz - 1) / 2 + 1;
    static const double w[3] = {0.25, 0.5, 0.25};
    memset(rc, 0, sizeof(double) * (size_t)cx * cy * cz);
#pragma omp parallel for schedule(static)
    for (int K = 1; K < cz - 1; ++K)
        for (int J = 1; J < cy - 1; ++J)
            for (int I = 1; I < cx - 1; ++I) {
                double s = 0.0;
                for (int dc = -1; dc <= 1; ++dc)
                    for (int db = -1; db <= 1; ++db)
                        for (int da = -1; da <= 1; ++da)
                            s += w[da + 1] * w[db + 1] * w[dc + 1] *
                                 r[I3(2 * I + da, 2 * J + db, 2 * K + dc)];
                rc[(size_t)I + (size_t)cx * ((size_t)J + (size_t)cy * (size_t)K)] = s;
            }
}

/* Trilinear prolongation + correction (reading C6):  u += P e_c at fine
 * interior nodes only.  Coincident node: e_c; edge midpoint: mean of 2; face centre: mean of 4;
 * cell centre: mean of 8 (tensor product of 1-D linear interpolation).  (nx,ny,nz) is FINE. */
void orc_prolong_add3(int nx, int ny, int nz, const double *ec, double *u)
{
    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1;
#pragma omp parallel for schedule(static)
    for (int k = 1; k < nz - 1; ++k)
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                int I0 = i / 2, I1 = (i + 1) / 2; /* equal when i is even */
                int J0 = j / 2, J1 = (j + 1) / 2;
                int K0 = k / 2, K1 = (k + 1) / 2;
                double s = 0.0;
                int Is[2] = {I0, I1}, Js[2] = {J0, J1}, Ks[2] = {K0, K1};
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a)
                            s += ec[(size_t)Is[a] + (size_t)cx * ((size_t)Js[b] + (size_t)cy * (size_t)Ks[c])];
                u[I3(i, j, k)] += 0.125 * s;
            }
}

/* sqrt( sum over interior nodes of r^2 )   (reading C10: unweighted l2, interior only) */
double orc_norm3(int nx, int ny, int nz, const double *r)
{
    double s = 0.0;
    for (int k = 1; k < nz - 1; ++k)
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                double v = r[I3(i, j, k)];
                s += v * v;
            }
    return sqrt(s);
}

/* || rhs - L u ||_2 over interior nodes. */
double orc_resnorm3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                    double alpha, const double *u, const double *rhs)
{
    double *r = (double *)malloc(sizeof(double) * (size_t)nx * ny * nz);
    orc_residual3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs, r);
    double n = orc_norm3(nx, ny, nz, r);
    free(r);
    return n;
}

/* Exact solve on one level (reading C9): the interior unknowns of  L u = rhs  with the
 * Dirichlet values found on the boundary nodes of u moved to the right-hand side; dense
 * Gaussian elimination with partial pivoting.  Unknown ordering: i fastest.  Returns 0 / -1. */
int orc_direct3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                double alpha, double *u, const double *rhs)
{
    int mx = nx - 2, my = ny - 2, mz = nz - 2;
    int n = mx * my * mz;
    double *A = (double *)calloc((size_t)n * n, sizeof(double));
    double *b = (double *)calloc((size_t)n, sizeof(double));
    if (!A || !b) { free(A); free(b); return -1; }
    for (int k = 1; k <= mz; ++k)
        for (int j = 1; j <= my; ++j)
            for (int i = 1; i <= mx; ++i) {
                int row = (i - 1) + mx * ((j - 1) + my * (k - 1));
                double ox = c[k] / (hx * hx), oy = c[k] / (hy * hy), oz = 1.0 / (hz * hz);
                A[(size_t)row * n + row] = diag3(hx, hy, hz, c[k], alpha);
                double bb = rhs ? rhs[I3(i, j, k)] : 0.0;
                int nb[6][3] = {{i - 1, j, k}, {i + 1, j, k}, {i, j - 1, k},
                                {i, j + 1, k}, {i, j, k - 1}, {i, j, k + 1}};
                double off[6] = {ox, ox, oy, oy, oz, oz};
                for (int q = 0; q < 6; ++q) {
                    int a = nb[q][0], bq = nb[q][1], cq = nb[q][2];
                    if (a >= 1 && a <= mx && bq >= 1 && bq <= my && cq >= 1 && cq <= mz)
                        A[(size_t)row * n + ((a - 1) + mx * ((bq - 1) + my * (cq - 1)))] = off[q];
                    else
                        bb -= off[q] * u[I3(a, bq, cq)];
                }
                b[row] = bb;
            }
    int rc = orc_dense_solve(n, A, b);
    if (rc == 0)
        for (int k = 1; k <= mz; ++k)
            for (int j = 1; j <= my; ++j)
                for (int i = 1; i <= mx; ++i)
                    u[I3(i, j, k)] = b[(i - 1) + mx * ((j - 1) + my * (k - 1))];
    free(A); free(b);
    return rc;
}

/* One V(n_pre,n_post) cycle on level `level` (SURVEY 8(c) "V(u,rhs,l)"), in place on u.
 * c is this level's coefficient table (nz entries); the next level's is injected,
 * c_{l+1}[K] = c_l[2K], and its operator rediscretised with 2h (readings C7, C8).
 * rhs may be NULL (== 0).  Returns 0, -1 if the coarse solve failed. */
int orc_vcycle3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                double alpha, double omega, int n_pre, int n_post, int level, int max_levels,
                double *u, const double *rhs)
{
    if (orc_is_coarsest(nx, ny, nz, level, max_levels))
        return orc_direct3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs);

    size_t N = (size_t)nx * ny * nz;
    double *tmp = (double *)malloc(sizeof(double) * N);
    double *r = (double *)malloc(sizeof(double) * N);
    for (int s = 0; s < n_pre; ++s) {
        orc_jacobi3(nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    orc_residual3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs, r);

    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1, cz = (nz - 1) / 2 + 1;
    size_t Nc = (size_t)cx * cy * cz;
    double *rc = (double *)malloc(sizeof(double) * Nc);
    double *ec = (double *)calloc(Nc, sizeof(double));
    double *cc = (double *)malloc(sizeof(double) * (size_t)cz);
    for (int K = 0; K < cz; ++K) cc[K] = c[2 * K];
    orc_restrict3(nx, ny, nz, r, rc);
    int st = orc_vcycle3(cx, cy, cz, 2.0 * hx, 2.0 * hy, 2.0 * hz, cc, alpha, omega, n_pre,
                         n_post, level + 1, max_levels, ec, rc);
    orc_prolong_add3(nx, ny, nz, ec, u);
    for (int s = 0; s < n_post; ++s) {
        orc_jacobi3(nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    free(tmp); free(r); free(rc); free(ec); free(cc);
    return st;
}

/* Generic 3D driver: repeat V-cycles on  L u = rhs  (Dirichlet data = boundary nodes of u)
 * until ||r_k|| <= tol * r0 or k == max_cycles (reading C10).  *r0_io <= 0 on entry: r0 is
 * the residual norm of the incoming iterate and is returned; otherwise the given r0 is used
 * (lets a caller continue cycle by cycle).  history[k] = ||r|| after cycle k+1 (up to
 * hist_len).  Returns the number of cycles done, or -1 on a failed coarse solve. */
int orc_solve3(int nx, int ny, int nz, double Lx, double Ly, double Lz, const double *c,
               double alpha, double omega, int n_pre, int n_post, int max_levels, double tol,
               int max_cycles, double *u, const double *rhs, double *r0_io, double *history,
               int hist_len)
{
    double hx = Lx / (nx - 1), hy = Ly / (ny - 1), hz = Lz / (nz - 1);
    double r0 = *r0_io;
    if (!(r0 > 0.0)) {
        r0 = orc_resnorm3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs);
        *r0_io = r0;
    }
    int k = 0;
    while (k < max_cycles) {
        if (orc_vcycle3(nx, ny, nz, hx, hy, hz, c, alpha, omega, n_pre, n_post, 0, max_levels, u, rhs))
            return -1;
        double rk = orc_resnorm3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs);
        if (k < hist_len) history[k] = rk;
        ++k;
        if (rk <= tol * r0) break;
    }
    return k;
}

/* Step 3 of the paper's procedure: eq (8) in the interior, rhs = 0, P = 0 on
 * the sides and top, P on the bottom plane as it stands in P.  c[k] = 1 + f[k]. */
int orc_solve_interior(int nx, int ny, int nz, double Lx, double Ly, double Lz, const double *f,
                       double alpha, double omega, int n_pre, int n_post, int max_levels,
                       double tol, int max_cycles, double *P, double *r0_io, double *history,
                       int hist_len)
{
    double *c = (double *)malloc(sizeof(double) * (size_t)nz);
    for (int k = 0; k < nz; ++k) c[k] = 1.0 + f[k];
    int n = orc_solve3(nx, ny, nz, Lx, Ly, Lz, c, alpha, omega, n_pre, n_post, max_levels, tol,
                       max_cycles, P, NULL, r0_io, history, hist_len);
    free(c);
    return n;
}

/* ====================================================================================
 *                                       2D
 *  (L2 u)_ij = (u_{i+1}-2u+u_{i-1})/hx^2 + (u_{j+1}-2u+u_{j-1})/hy^2,  eq (11)
 * ================================================================================== */

void orc_apply2(int nx, int ny, double hx, double hy, const double *u, double *out)
{
    memset(out, 0, sizeof(double) * (size_t)nx * ny);
#pragma omp parallel for schedule(static)
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) {
            double uc = u[I2(i, j)];
            double dxx = (u[I2(i + 1, j)] - 2.0 * uc + u[I2(i - 1, j)]) / (hx * hx);
            double dyy = (u[I2(i, j + 1)] - 2.0 * uc + u[I2(i, j - 1)]) / (hy * hy);
            out[I2(i, j)] = dxx + dyy;
        }
}

void orc_residual2(int nx, int ny, double hx, double hy, const double *u, const double *rhs, double *r)
{
    orc_apply2(nx, ny, hx, hy, u, r);
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) {
            size_t p = I2(i, j);
            r[p] = (rhs ? rhs[p] : 0.0) - r[p];
        }
}

/* Weighted Gauss-Jacobi for eq (11): the kernel the paper describes. */
void orc_jacobi2(int nx, int ny, double hx, double hy, double omega, const double *u,
                 const double *rhs, double *unew)
{
    double D = -2.0 / (hx * hx) - 2.0 / (hy * hy);
    memcpy(unew, u, sizeof(double) * (size_t)nx * ny); /* boundary branch */
#pragma omp parallel for schedule(static)
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) {
            size_t p = I2(i, j);
            double uc = u[p];
            double dxx = (u[I2(i + 1, j)] - 2.0 * uc + u[I2(i - 1, j)]) / (hx * hx);
            double dyy = (u[I2(i, j + 1)] - 2.0 * uc + u[I2(i, j - 1)]) / (hy * hy);
            unew[p] = uc + (omega / D) * ((rhs ? rhs[p] : 0.0) - (dxx + dyy));
        }
}

/* 9-point full weighting, w = (1/4,1/2,1/4) per axis.  (nx,ny) is the FINE grid. */
void orc_restrict2(int nx, int ny, const double *r, double *rc)
{
    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1;
    static const double w[3] = {0.25, 0.5, 0.25};
    memset(rc, 0, sizeof(double) * (size_t)cx * cy);
    for (int J = 1; J < cy - 1; ++J)
        for (int I = 1; I < cx - 1; ++I) {
            double s = 0.0;
            for (int db = -1; db <= 1; ++db)
                for (int da = -1; da <= 1; ++da)
                    s += w[da + 1] * w[db + 1] * r[I2(2 * I + da, 2 * J + db)];
            rc[(size_t)I + (size_t)cx * (size_t)J] = s;
        }
}

/* Bilinear prolongation + correction at fine interior nodes.  (nx,ny) is FINE. */
void orc_prolong_add2(int nx, int ny, const double *ec, double *u)
{
    int cx = (nx - 1) / 2 + 1;
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) {
            int Is[2] = {i / 2, (i + 1) / 2}, Js[2] = {j / 2, (j + 1) / 2};
            double s = 0.0;
            for (int b = 0; b < 2; ++b)
                for (int a = 0; a < 2; ++a) s += ec[(size_t)Is[a] + (size_t)cx * (size_t)Js[b]];
            u[I2(i, j)] += 0.25 * s;
        }
}

double orc_norm2(int nx, int ny, const double *r)
{
    double s = 0.0;
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) {
            double v = r[I2(i, j)];
            s += v * v;
        }
    return sqrt(s);
}

double orc_resnorm2(int nx, int ny, double hx, double hy, const double *u, const double *rhs)
{
    double *r = (double *)malloc(sizeof(double) * (size_t)nx * ny);
    orc_residual2(nx, ny, hx, hy, u, rhs, r);
    double n = orc_norm2(nx, ny, r);
    free(r);
    return n;
}

int orc_direct2(int nx, int ny, double hx, double hy, double *u, const double *rhs)
{
    int mx = nx - 2, my = ny - 2, n = mx * my;
    double *A = (double *)calloc((size_t)n * n, sizeof(double));
    double *b = (double *)calloc((size_t)n, sizeof(double));
    if (!A || !b) { free(A); free(b); return -1; }
    double ox = 1.0 / (hx * hx), oy = 1.0 / (hy * hy);
    for (int j = 1; j <= my; ++j)
        for (int i = 1; i <= mx; ++i) {
            int row = (i - 1) + mx * (j - 1);
            A[(size_t)row * n + row] = -2.0 * ox - 2.0 * oy;
            double bb = rhs ? rhs[I2(i, j)] : 0.0;
            int nb[4][2] = {{i - 1, j}, {i + 1, j}, {i, j - 1}, {i, j + 1}};
            double off[4] = {ox, ox, oy, oy};
            for (int q = 0; q < 4; ++q) {
                int a = nb[q][0], bq = nb[q][1];
                if (a >= 1 && a <= mx && bq >= 1 && bq <= my)
                    A[(size_t)row * n + ((a - 1) + mx * (bq - 1))] = off[q];
                else
                    bb -= off[q] * u[I2(a, bq)];
            }
            b[row] = bb;
        }
    int rc = orc_dense_solve(n, A, b);
    if (rc == 0)
        for (int j = 1; j <= my; ++j)
            for (int i = 1; i <= mx; ++i) u[I2(i, j)] = b[(i - 1) + mx * (j - 1)];
    free(A); free(b);
    return rc;
}

int orc_vcycle2(int nx, int ny, double hx, double hy, double omega, int n_pre, int n_post,
                int level, int max_levels, double *u, const double *rhs)
{
    if (orc_is_coarsest(nx, ny, 1, level, max_levels)) return orc_direct2(nx, ny, hx, hy, u, rhs);
    size_t N = (size_t)nx * ny;
    double *tmp = (double *)malloc(sizeof(double) * N);
    double *r = (double *)malloc(sizeof(double) * N);
    for (int s = 0; s < n_pre; ++s) {
        orc_jacobi2(nx, ny, hx, hy, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    orc_residual2(nx, ny, hx, hy, u, rhs, r);
    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1;
    double *rc = (double *)malloc(sizeof(double) * (size_t)cx * cy);
    double *ec = (double *)calloc((size_t)cx * cy, sizeof(double));
    orc_restrict2(nx, ny, r, rc);
    int st = orc_vcycle2(cx, cy, 2.0 * hx, 2.0 * hy, omega, n_pre, n_post, level + 1, max_levels, ec, rc);
    orc_prolong_add2(nx, ny, ec, u);
    for (int s = 0; s < n_post; ++s) {
        orc_jacobi2(nx, ny, hx, hy, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    free(tmp); free(r); free(rc); free(ec);
    return st;
}

int orc_solve2(int nx, int ny, double Lx, double Ly, double omega, int n_pre, int n_post,
               int max_levels, double tol, int max_cycles, double *u, const double *rhs,
               double *r0_io, double *history, int hist_len)
{
    double hx = Lx / (nx - 1), hy = Ly / (ny - 1);
    double r0 = *r0_io;
    if (!(r0 > 0.0)) {
        r0 = orc_resnorm2(nx, ny, hx, hy, u, rhs);
        *r0_io = r0;
    }
    int k = 0;
    while (k < max_cycles) {
        if (orc_vcycle2(nx, ny, hx, hy, omega, n_pre, n_post, 0, max_levels, u, rhs)) return -1;
        double rk = orc_resnorm2(nx, ny, hx, hy, u, rhs);
        if (k < hist_len) history[k] = rk;
        ++k;
        if (rk <= tol * r0) break;
    }
    return k;
}

/* Steps 1-2 of the paper's procedure: u2 = 0, rhs2 = -Bz0 at interior (i,j),
 * edges of u2 stay 0; V-cycles to boundary_tol.  u2 (nx*ny) is the output: P(x,y,0). */
int orc_solve_boundary(int nx, int ny, double Lx, double Ly, const double *Bz0, double omega,
                       int n_pre, int n_post, int max_levels, double tol, int max_cycles,
                       double *u2, double *r0_out, double *history, int hist_len)
{
    size_t N = (size_t)nx * ny;
    double *rhs = (double *)calloc(N, sizeof(double));
    memset(u2, 0, sizeof(double) * N);
    for (int j = 1; j < ny - 1; ++j)
        for (int i = 1; i < nx - 1; ++i) rhs[I2(i, j)] = -Bz0[I2(i, j)];
    *r0_out = 0.0;
    int n = orc_solve2(nx, ny, Lx, Ly, omega, n_pre, n_post, max_levels, tol, max_cycles, u2, rhs,
                       r0_out, history, hist_len);
    free(rhs);
    return n;
}

/* ====================================================================================
 *  Field recovery (eq 5 with T = alpha P; eqs 9, 10; readings C13-C15)
 *    Bz = -(dxx + dyy) P                         (eq 11 applied at every z)
 *    Bx =  alpha D_y P + D_x D_z P
 *    By = -alpha D_x P + D_y D_z P
 *    p   = p_b - xi Bz^2/(2 mu0)                                            (eq 9)
 *    rho = rho_b + (1/g) [ xi' Bz^2/(2 mu0) + (1/mu0) xi B . grad Bz ]      (eq 10)
 *  with xi = -f, xi' = -f' (C1).  D = central first difference, dxx = compact second
 *  difference.  Side and top boundary nodes: B = 0, p = p_b, rho = rho_b.
 *  Bottom plane k = 0 at interior (i,j): D_z is the one-sided 2nd-order
 *  (-3 u_0 + 4 u_1 - u_2)/(2 hz).  grad Bz uses the Bz array just built (zeros on sides/top).
 *  dfdz == NULL: central FD of the f samples, one-sided 2nd-order at k = 0 and nz-1 (C14).
 * ================================================================================== */
static double dz_at(const double *a, int nx, int ny, int nz, int i, int j, int k, double hz)
{
    if (k == 0)
        return (-3.0 * a[I3(i, j, 0)] + 4.0 * a[I3(i, j, 1)] - a[I3(i, j, 2)]) / (2.0 * hz);
    (void)nz;
    return (a[I3(i, j, k + 1)] - a[I3(i, j, k - 1)]) / (2.0 * hz);
}

void orc_fields(int nx, int ny, int nz, double Lx, double Ly, double Lz, double alpha,
                const double *f, const double *dfdz, const double *p_b, const double *rho_b,
                double mu0, double g, const double *P, double *Bx, double *By, double *Bz,
                double *p, double *rho)
{
    double hx = Lx / (nx - 1), hy = Ly / (ny - 1), hz = Lz / (nz - 1);
    size_t N = (size_t)nx * ny * nz;
    memset(Bx, 0, sizeof(double) * N);
    memset(By, 0, sizeof(double) * N);
    memset(Bz, 0, sizeof(double) * N);

    /* B at every node that is not on a side or on the top: k = 0 .. nz-2, interior (i,j). */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz - 1; ++k)
        for (int j = 1; j < ny - 1; ++j)
            for (int i = 1; i < nx - 1; ++i) {
                size_t q = I3(i, j, k);
                double uc = P[q];
                double dxx = (P[I3(i + 1, j, k)] - 2.0 * uc + P[I3(i - 1, j, k)]) / (hx * hx);
                double dyy = (P[I3(i, j + 1, k)] - 2.0 * uc + P[I3(i, j - 1, k)]) / (hy * hy);
                double dxP = (P[I3(i + 1, j, k)] - P[I3(i - 1, j, k)]) / (2.0 * hx);
                double dyP = (P[I3(i, j + 1, k)] - P[I3(i, j - 1, k)]) / (2.0 * hy);
                double dxdz = (dz_at(P, nx, ny, nz, i + 1, j, k, hz) - dz_at(P, nx, ny, nz, i - 1, j, k, hz)) / (2.0 * hx);
                double dydz = (dz_at(P, nx, ny, nz, i, j + 1, k, hz) - dz_at(P, nx, ny, nz, i, j - 1, k, hz)) / (2.0 * hy);
                Bz[q] = -(dxx + dyy);
                Bx[q] = alpha * dyP + dxdz;
                By[q] = -alpha * dxP + dydz;
            }

    /* p and rho. */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k) {
        double fk = f[k], dfk;
        if (dfdz) dfk = dfdz[k];
        else if (k == 0) dfk = (-3.0 * f[0] + 4.0 * f[1] - f[2]) / (2.0 * hz);
        else if (k == nz - 1) dfk = (3.0 * f[nz - 1] - 4.0 * f[nz - 2] + f[nz - 3]) / (2.0 * hz);
        else dfk = (f[k + 1] - f[k - 1]) / (2.0 * hz);
        double xi = -fk, dxi = -dfk;
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t q = I3(i, j, k);
                int wall = (i == 0 || i == nx - 1 || j == 0 || j == ny - 1 || k == nz - 1);
                if (wall) { p[q] = p_b[k]; rho[q] = rho_b[k]; continue; }
                double bz = Bz[q];
                double dxBz = (Bz[I3(i + 1, j, k)] - Bz[I3(i - 1, j, k)]) / (2.0 * hx);
                double dyBz = (Bz[I3(i, j + 1, k)] - Bz[I3(i, j - 1, k)]) / (2.0 * hy);
                double dzBz = dz_at(Bz, nx, ny, nz, i, j, k, hz);
                p[q] = p_b[k] - xi * bz * bz / (2.0 * mu0);
                rho[q] = rho_b[k] + (1.0 / g) * (dxi * bz * bz / (2.0 * mu0) +
                                                 (1.0 / mu0) * xi * (Bx[q] * dxBz + By[q] * dyBz + bz * dzBz));
            }
    }
}

/* ------------------------------------------------------------------------------------
 * Diagnostics of a computed equilibrium (the quantities of the paper's Figs 2, 4-7,
 * PAPER.md:164-196): |B| and the current density  j = curl B / mu0  (eq 2) with |j|.
 * Second-order central differences of the B that orc_fields returns ("derivatives must be dealt with
 * using finite differences"); on the bottom plane the z-derivatives are the one-sided second-order ones, as for B
 * itself (C13); on the side and top boundary nodes, where B = 0 is imposed, j is set to 0.
 * ---------------------------------------------------------------------------------- */
void orc_diagnostics(int nx, int ny, int nz, double Lx, double Ly, double Lz, double mu0,
                     const double *Bx, const double *By, const double *Bz,
                     double *absB, double *jx, double *jy, double *jz, double *absJ)
{
    double hx = Lx / (nx - 1), hy = Ly / (ny - 1), hz = Lz / (nz - 1);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t q = I3(i, j, k);
                absB[q] = sqrt(Bx[q] * Bx[q] + By[q] * By[q] + Bz[q] * Bz[q]);
                int wall = (i == 0 || i == nx - 1 || j == 0 || j == ny - 1 || k == nz - 1);
                if (wall) { jx[q] = jy[q] = jz[q] = absJ[q] = 0.0; continue; }
                double dyBz = (Bz[I3(i, j + 1, k)] - Bz[I3(i, j - 1, k)]) / (2.0 * hy);
                double dxBz = (Bz[I3(i + 1, j, k)] - Bz[I3(i - 1, j, k)]) / (2.0 * hx);
                double dxBy = (By[I3(i + 1, j, k)] - By[I3(i - 1, j, k)]) / (2.0 * hx);
                double dyBx = (Bx[I3(i, j + 1, k)] - Bx[I3(i, j - 1, k)]) / (2.0 * hy);
                double dzBy = dz_at(By, nx, ny, nz, i, j, k, hz);
                double dzBx = dz_at(Bx, nx, ny, nz, i, j, k, hz);
                double a = (dyBz - dzBy) / mu0, b = (dzBx - dxBz) / mu0, c = (dxBy - dyBx) / mu0;
                jx[q] = a; jy[q] = b; jz[q] = c;
                absJ[q] = sqrt(a * a + b * b + c * c);
            }
}

/* ------------------------------------------------------------------------------------
 * Field-line integration (SURVEY 8(f) NEXT-4; the field lines of the paper's Figs 1, 4, 5, PAPER.md:142-144, :158-186;
 * the paper draws them with IDL, and names no integrator -- reading C24 in DESIGN.md):
 *     dx/ds = dir * B(x) / |B(x)|          (s = arc length, dir = +1 / -1)
 * B(x) between the nodes = trilinear interpolation of the nodal B that orc_fields returns; classical fourth-order
 * Runge-Kutta with a fixed arc-length step `step`.  Point 0 is the seed; a line ends when a Runge-Kutta stage or the new
 * point falls outside the box [0,Lx]x[0,Ly]x[0,Lz], when |B| <= bmin at a stage (a null), or at max_points.
 * A seed outside the box gives 0 points.  lines: nseeds x max_points x 3 (x, y, z), points beyond npoints[s] untouched.
 * Every product-sum is written with fma() in the order the formulas below show, so that an implementation that does the
 * same gets the same points bit for bit (the exit tests decide an integer).
 * ---------------------------------------------------------------------------------- */
static int fl_inside(double x, double y, double z, double Lx, double Ly, double Lz)
{
    return x >= 0.0 && x <= Lx && y >= 0.0 && y <= Ly && z >= 0.0 && z <= Lz;
}

/* trilinear sample of one component a at (x,y,z): cell (i,j,k) = floor(x/hx) clamped to [0, n-2], weights t = x/hx - i;
 * lerp along x, then y, then z, each as fma(t, b - a, a) */
static double fl_sample(const double *a, int nx, int ny, int nz, double ihx, double ihy, double ihz,
                        double x, double y, double z)
{
    double fx = x * ihx, fy = y * ihy, fz = z * ihz;
    int i = (int)floor(fx), j = (int)floor(fy), k = (int)floor(fz);
    if (i < 0) i = 0; if (i > nx - 2) i = nx - 2;
    if (j < 0) j = 0; if (j > ny - 2) j = ny - 2;
    if (k < 0) k = 0; if (k > nz - 2) k = nz - 2;
    double tx = fx - i, ty = fy - j, tz = fz - k;
    double a000 = a[I3(i, j, k)], a100 = a[I3(i + 1, j, k)], a010 = a[I3(i, j + 1, k)], a110 = a[I3(i + 1, j + 1, k)];
    double a001 = a[I3(i, j, k + 1)], a101 = a[I3(i + 1, j, k + 1)], a011 = a[I3(i, j + 1, k + 1)], a111 = a[I3(i + 1, j + 1, k + 1)];
    double b00 = fma(tx, a100 - a000, a000), b10 = fma(tx, a110 - a010, a010);
    double b01 = fma(tx, a101 - a001, a001), b11 = fma(tx, a111 - a011, a011);
    double c0 = fma(ty, b10 - b00, b00), c1 = fma(ty, b11 - b01, b01);
    return fma(tz, c1 - c0, c0);
}

/* unit tangent dir*B/|B| at (x,y,z); returns 0 if outside the box or |B| <= bmin */
static int fl_tangent(const double *Bx, const double *By, const double *Bz, int nx, int ny, int nz, double Lx, double Ly,
                      double Lz, double ihx, double ihy, double ihz, double dir, double bmin, double x, double y, double z,
                      double *t)
{
    if (!fl_inside(x, y, z, Lx, Ly, Lz)) return 0;
    double bx = fl_sample(Bx, nx, ny, nz, ihx, ihy, ihz, x, y, z);
    double by = fl_sample(By, nx, ny, nz, ihx, ihy, ihz, x, y, z);
    double bz = fl_sample(Bz, nx, ny, nz, ihx, ihy, ihz, x, y, z);
    double m = sqrt(fma(bz, bz, fma(by, by, bx * bx)));
    if (!(m > bmin)) return 0;
    double s = dir / m;
    t[0] = bx * s; t[1] = by * s; t[2] = bz * s;
    return 1;
}

void orc_fieldlines(int nx, int ny, int nz, double Lx, double Ly, double Lz, const double *Bx, const double *By,
                    const double *Bz, int nseeds, const double *seeds, double step, int max_points, int direction,
                    double bmin, double *lines, int *npoints)
{
    double ihx = (nx - 1) / Lx, ihy = (ny - 1) / Ly, ihz = (nz - 1) / Lz;
    double dir = direction < 0 ? -1.0 : 1.0, h = step, h2 = 0.5 * step, h6 = step / 6.0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int s = 0; s < nseeds; ++s) {
        double x = seeds[3 * s], y = seeds[3 * s + 1], z = seeds[3 * s + 2];
        double *out = lines + (size_t)s * max_points * 3;
        int n = 0;
        if (max_points > 0 && fl_inside(x, y, z, Lx, Ly, Lz)) {
            out[0] = x; out[1] = y; out[2] = z;
            n = 1;
            while (n < max_points) {
                double k1[3], k2[3], k3[3], k4[3];
                if (!fl_tangent(Bx, By, Bz, nx, ny, nz, Lx, Ly, Lz, ihx, ihy, ihz, dir, bmin, x, y, z, k1)) break;
                if (!fl_tangent(Bx, By, Bz, nx, ny, nz, Lx, Ly, Lz, ihx, ihy, ihz, dir, bmin, fma(h2, k1[0], x), fma(h2, k1[1], y), fma(h2, k1[2], z), k2)) break;
                if (!fl_tangent(Bx, By, Bz, nx, ny, nz, Lx, Ly, Lz, ihx, ihy, ihz, dir, bmin, fma(h2, k2[0], x), fma(h2, k2[1], y), fma(h2, k2[2], z), k3)) break;
                if (!fl_tangent(Bx, By, Bz, nx, ny, nz, Lx, Ly, Lz, ihx, ihy, ihz, dir, bmin, fma(h, k3[0], x), fma(h, k3[1], y), fma(h, k3[2], z), k4)) break;
                double xn = fma(h6, (k1[0] + k4[0]) + 2.0 * (k2[0] + k3[0]), x);
                double yn = fma(h6, (k1[1] + k4[1]) + 2.0 * (k2[1] + k3[1]), y);
                double zn = fma(h6, (k1[2] + k4[2]) + 2.0 * (k2[2] + k3[2]), z);
                if (!fl_inside(xn, yn, zn, Lx, Ly, Lz)) break;
                x = xn; y = yn; z = zn;
                out[3 * n] = x; out[3 * n + 1] = y; out[3 * n + 2] = z;
                ++n;
            }
        }
        npoints[s] = n;
    }
}

/* ====================================================================================
 *  Solver variants inside "a multigrid method" (SURVEY 8(f) NEXT-3; PAPER.md:90 "multigrid methods", :148-156: the
 *  paper's xi_2 profile takes 1 - xi down to 0.05 near the base, where the z-coupling of eq (8) dominates the horizontal
 *  one and point relaxation smooths poorly).  These change the iterates, so they are options with their own pins; the
 *  functions above are untouched.  Readings C25-C27 in DESIGN.md.
 * ================================================================================== */

/* One weighted z-LINE Jacobi sweep (reading C25).  Split L = T + O: T couples a node to itself and to its two z-neighbours,
 *     (T u)_ijk = (u_{k+1} + u_{k-1})/hz^2 + D_k u_k,      D_k the diagonal of L on plane k,
 * O is the rest (the four horizontal neighbours).  All lines are relaxed simultaneously from the old values (two arrays,
 * as the paper's Jacobi):   unew = u + omega * d,   T d = rhs - L u  on every line (i,j), d = 0 at k = 0, nz-1.
 * T is the same tridiagonal matrix for every line; it is solved by the Thomas algorithm (no pivoting: |D_k| > 2/hz^2
 * whenever the operator is definite).  Boundary nodes: unew = u. */
void orc_zline3(int nx, int ny, int nz, double hx, double hy, double hz, const double *c,
                double alpha, double omega, const double *u, const double *rhs, double *unew)
{
    size_t N = (size_t)nx * ny * nz;
    int m = nz - 2;
    double a = 1.0 / (hz * hz);
    double *r = (double *)malloc(sizeof(double) * N);
    orc_residual3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs, r);
    memcpy(unew, u, sizeof(double) * N); /* boundary branch */
#pragma omp parallel for schedule(static)
    for (int j = 1; j < ny - 1; ++j) {
        double *cp = (double *)malloc(sizeof(double) * (size_t)(m + 2));
        double *dp = (double *)malloc(sizeof(double) * (size_t)(m + 2));
        for (int i = 1; i < nx - 1; ++i) {
            /* forward elimination, k = 1 .. nz-2 */
            double den = diag3(hx, hy, hz, c[1], alpha);
            cp[1] = a / den;
            dp[1] = r[I3(i, j, 1)] / den;
            for (int k = 2; k <= m; ++k) {
                den = diag3(hx, hy, hz, c[k], alpha) - a * cp[k - 1];
                cp[k] = a / den;
                dp[k] = (r[I3(i, j, k)] - a * dp[k - 1]) / den;
            }
            /* back substitution */
            double d = dp[m];
            unew[I3(i, j, m)] = u[I3(i, j, m)] + omega * d;
            for (int k = m - 1; k >= 1; --k) {
                d = dp[k] - cp[k] * d;
                unew[I3(i, j, k)] = u[I3(i, j, k)] + omega * d;
            }
        }
        free(cp); free(dp);
    }
    free(r);
}

/* One smoothing sweep by name: 0 = point Jacobi (orc_jacobi3), 1 = z-line Jacobi (orc_zline3). */
static void smooth3(int smoother, int nx, int ny, int nz, double hx, double hy, double hz, const double *c, double alpha,
                    double omega, const double *u, const double *rhs, double *unew)
{
    if (smoother == 1) orc_zline3(nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, unew);
    else orc_jacobi3(nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, unew);
}

/* orc_vcycle3 with the smoother as an option (the same steps in the same order; smoother = 0 reproduces it). */
int orc_vcycle3s(int nx, int ny, int nz, double hx, double hy, double hz, const double *c, double alpha, double omega,
                 int n_pre, int n_post, int level, int max_levels, int smoother, double *u, const double *rhs)
{
    if (orc_is_coarsest(nx, ny, nz, level, max_levels))
        return orc_direct3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs);
    size_t N = (size_t)nx * ny * nz;
    double *tmp = (double *)malloc(sizeof(double) * N);
    double *r = (double *)malloc(sizeof(double) * N);
    for (int s = 0; s < n_pre; ++s) {
        smooth3(smoother, nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    orc_residual3(nx, ny, nz, hx, hy, hz, c, alpha, u, rhs, r);
    int cx = (nx - 1) / 2 + 1, cy = (ny - 1) / 2 + 1, cz = (nz - 1) / 2 + 1;
    size_t Nc = (size_t)cx * cy * cz;
    double *rc = (double *)malloc(sizeof(double) * Nc);
    double *ec = (double *)calloc(Nc, sizeof(double));
    double *cc = (double *)malloc(sizeof(double) * (size_t)cz);
    for (int K = 0; K < cz; ++K) cc[K] = c[2 * K];
    orc_restrict3(nx, ny, nz, r, rc);
    int st = orc_vcycle3s(cx, cy, cz, 2.0 * hx, 2.0 * hy, 2.0 * hz, cc, alpha, omega, n_pre, n_post, level + 1, max_levels,
                          smoother, ec, rc);
    orc_prolong_add3(nx, ny, nz, ec, u);
    for (int s = 0; s < n_post; ++s) {
        smooth3(smoother, nx, ny, nz, hx, hy, hz, c, alpha, omega, u, rhs, tmp);
        memcpy(u, tmp, sizeof(double) * N);
    }
    free(tmp); free(r); free(rc); free(ec); free(cc);
    return st;
}

/* Full-multigrid start (reading C26): the interior of P (bottom plane = data, as for orc_solve_interior) is replaced by
 * an initial guess built from the coarse grids upwards instead of zero:
 *   level l carries the bottom data by injection, P_l(I,J,0) = P(2^l I, 2^l J, 0), zero on sides and top;
 *   coarsest level: exact solve;   level l < coarsest: u_l = trilinear interpolation of u_{l+1} at the interior nodes
 *   (its bottom plane is the injected data), followed by n_fmg V-cycles of eq (8) on level l (rhs = 0).
 * Level 0 included: on return P is the FMG iterate; the caller goes on with ordinary V-cycles.  Returns 0 / -1. */
int orc_fmg_interior(int nx, int ny, int nz, double Lx, double Ly, double Lz, const double *f, double alpha, double omega,
                     int n_pre, int n_post, int max_levels, int smoother, int n_fmg, double *P)
{
    int lnx[32], lny[32], lnz[32], nl = 0;
    {
        int ax = nx, ay = ny, az = nz;
        for (;;) {
            lnx[nl] = ax; lny[nl] = ay; lnz[nl] = az;
            ++nl;
            if (orc_is_coarsest(ax, ay, az, nl - 1, max_levels)) break;
            ax = (ax - 1) / 2 + 1; ay = (ay - 1) / 2 + 1; az = (az - 1) / 2 + 1;
        }
    }
    double *cl[32], *ul[32];
    for (int l = 0; l < nl; ++l) {
        int s = 1 << l;
        cl[l] = (double *)malloc(sizeof(double) * (size_t)lnz[l]);
        for (int K = 0; K < lnz[l]; ++K) cl[l][K] = 1.0 + f[(size_t)s * K];
        ul[l] = (double *)calloc((size_t)lnx[l] * lny[l] * lnz[l], sizeof(double));
        for (int J = 0; J < lny[l]; ++J)
            for (int I = 0; I < lnx[l]; ++I)
                ul[l][(size_t)I + (size_t)lnx[l] * J] = P[(size_t)(s * I) + (size_t)nx * (size_t)(s * J)];
    }
    int st = 0;
    for (int l = nl - 1; l >= 0 && st == 0; --l) {
        double s = (double)(1 << l);
        double hx = s * Lx / (nx - 1), hy = s * Ly / (ny - 1), hz = s * Lz / (nz - 1);
        if (l == nl - 1) {
            st = orc_direct3(lnx[l], lny[l], lnz[l], hx, hy, hz, cl[l], alpha, ul[l], NULL);
        } else {
            orc_prolong_add3(lnx[l], lny[l], lnz[l], ul[l + 1], ul[l]); /* interior of ul[l] is zero: this IS interpolation */
            for (int q = 0; q < n_fmg && st == 0; ++q)
                st = orc_vcycle3s(lnx[l], lny[l], lnz[l], hx, hy, hz, cl[l], alpha, omega, n_pre, n_post, l, max_levels,
                                  smoother, ul[l], NULL);
        }
    }
    memcpy(P, ul[0], sizeof(double) * (size_t)nx * ny * nz);
    for (int l = 0; l < nl; ++l) { free(cl[l]); free(ul[l]); }
    return st;
}

/* orc_solve_interior with the variants as options: smoother (0 point, 1 z-line Jacobi) and fmg (0: start from the zero
 * interior as the paper's step 1 says;  n > 0: full-multigrid start with n V-cycles per level).  r0 is ALWAYS
 * the residual norm of the zero-interior iterate (bottom data only), so tolerances mean the same with and without FMG. */
int orc_solve_interior_opt(int nx, int ny, int nz, double Lx, double Ly, double Lz, const double *f, double alpha,
                           double omega, int n_pre, int n_post, int max_levels, int smoother, int fmg, double tol,
                           int max_cycles, double *P, double *r0_io, double *history, int hist_len)
{
    double hx = Lx / (nx - 1), hy = Ly / (ny - 1), hz = Lz / (nz - 1);
    double *c = (double *)malloc(sizeof(double) * (size_t)nz);
    for (int k = 0; k < nz; ++k) c[k] = 1.0 + f[k];
    double r0 = *r0_io;
    if (!(r0 > 0.0)) {
        r0 = orc_resnorm3(nx, ny, nz, hx, hy, hz, c, alpha, P, NULL);
        *r0_io = r0;
    }
    int k = 0;
    if (fmg > 0) {
        if (orc_fmg_interior(nx, ny, nz, Lx, Ly, Lz, f, alpha, omega, n_pre, n_post, max_levels, smoother, fmg, P)) { free(c); return -1; }
        /* the FMG iterate may already meet the tolerance: history[-] has no slot for it, so it is reported through a cycle
         * count of 0 only if it does */
        if (orc_resnorm3(nx, ny, nz, hx, hy, hz, c, alpha, P, NULL) <= tol * r0) { free(c); return 0; }
    }
    while (k < max_cycles) {
        if (orc_vcycle3s(nx, ny, nz, hx, hy, hz, c, alpha, omega, n_pre, n_post, 0, max_levels, smoother, P, NULL)) { free(c); return -1; }
        double rk = orc_resnorm3(nx, ny, nz, hx, hy, hz, c, alpha, P, NULL);
        if (k < hist_len) history[k] = rk;
        ++k;
        if (rk <= tol * r0) break;
    }
    free(c);
    return k;
}
