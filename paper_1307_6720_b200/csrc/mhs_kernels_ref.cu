// Reference kernels of libmhs_b200: one thread per node, one kernel per multigrid component, global
// memory only -- the design the paper describes for its Gauss-Jacobi kernel (one
// thread per node, flat array with neighbours at off+-1 / off+-DIM, one branch for boundary nodes,
// read d_P1 / write d_P2) carried over to all four components of PAPER.md:210.  They run every level
// that has no tuned kernel, all 2D work, and everything when MHS_FLAG_REFERENCE_KERNELS is set
// (A/B baseline for the tuned kernels in mhs_kernels_fast.cu).
#include "mhs_device.cuh"

namespace mhs {

// ------------------------------------------------------------------------------------------------
// Weighted Gauss-Jacobi sweep (C4, C12): interior nodes
//   out = u + (omega/D_k) (rhs - L u),   boundary nodes are never written (they stay 0 / data).
// ------------------------------------------------------------------------------------------------
template <typename T, bool D3>
__global__ void __launch_bounds__(256) k_smooth_ref(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs,
                                                     T* __restrict__ out, const int* __restrict__ done)
{
    if (done && *done) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = D3 ? (int)blockIdx.z + 1 : 0;
    if (i >= p.sx || j >= p.sy || i == 0 || j == 0) return;
    const long long c = i + (long long)p.sx * j + p.sp * k;
    const T lu = apply_L<T, D3>(p, u, c, k);
    const T f = rhs ? rhs[c] : T(0);
    out[c] = u[c] + p.tab[3 * p.nz + k] * (f - lu);
}

// r = rhs - L u at interior nodes ("calculation of the residual").
template <typename T, bool D3>
__global__ void __launch_bounds__(256) k_residual_ref(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs,
                                                       T* __restrict__ r, const int* __restrict__ done)
{
    if (done && *done) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = D3 ? (int)blockIdx.z + 1 : 0;
    if (i >= p.sx || j >= p.sy || i == 0 || j == 0) return;
    const long long c = i + (long long)p.sx * j + p.sp * k;
    const T f = rhs ? rhs[c] : T(0);
    r[c] = f - apply_L<T, D3>(p, u, c, k);
}

// Full weighting ("reduction"; C6): coarse interior node (I,J,K) <- 27 (9) fine nodes.
template <typename T, bool D3>
__global__ void __launch_bounds__(256) k_restrict_ref(int fsx, long long fsp, const T* __restrict__ r, int csx, int csy,
                                                       long long csp, T* __restrict__ rc, const int* __restrict__ done)
{
    if (done && *done) return;
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = D3 ? (int)blockIdx.z + 1 : 0;
    if (I >= csx || J >= csy || I == 0 || J == 0) return;
    const T* q = r + 2 * I + (long long)fsx * (2 * J) + fsp * (2 * K);
    T s = T(0);
#pragma unroll
    for (int dc = (D3 ? -1 : 0); dc <= (D3 ? 1 : 0); ++dc) {
        T sp = T(0);
#pragma unroll
        for (int db = -1; db <= 1; ++db) {
            const T* row = q + (long long)fsx * db + fsp * dc;
            const T sx = T(0.25) * (row[-1] + row[1]) + T(0.5) * row[0];
            sp += (db == 0 ? T(0.5) : T(0.25)) * sx;
        }
        s += (D3 ? (dc == 0 ? T(0.5) : T(0.25)) : T(1)) * sp;
    }
    rc[I + (long long)csx * J + csp * K] = s;
}

// Tri/bi-linear prolongation + correction at fine interior nodes (C6).
template <typename T, bool D3>
__global__ void __launch_bounds__(256) k_prolong_ref(int fsx, int fsy, long long fsp, T* __restrict__ u, int csx,
                                                      long long csp, const T* __restrict__ ec, const int* __restrict__ done)
{
    if (done && *done) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = D3 ? (int)blockIdx.z + 1 : 0;
    if (i >= fsx || j >= fsy || i == 0 || j == 0) return;
    const int I0 = i >> 1, I1 = (i + 1) >> 1, J0 = j >> 1, J1 = (j + 1) >> 1;
    const int K0 = k >> 1, K1 = (k + 1) >> 1;
    const T* a = ec + csp * K0;
    T s = (a[I0 + (long long)csx * J0] + a[I1 + (long long)csx * J0]) +
          (a[I0 + (long long)csx * J1] + a[I1 + (long long)csx * J1]);
    if (D3) {
        const T* b = ec + csp * K1;
        s += (b[I0 + (long long)csx * J0] + b[I1 + (long long)csx * J0]) +
             (b[I0 + (long long)csx * J1] + b[I1 + (long long)csx * J1]);
    }
    const long long c = i + (long long)fsx * j + fsp * k;
    u[c] += (D3 ? T(0.125) : T(0.25)) * s;
}

// Exact coarsest-level solve (C9): e = A^{-1} rhs over the interior unknowns, A^{-1} precomputed on
// the host in fp64 by Gauss-Jordan with partial pivoting (mhs_create).  One block.
template <typename T>
__global__ void k_coarse_solve(int mx, int my, int mz, int sx, long long sp, int k0, const T* __restrict__ ainv,
                               const T* __restrict__ rhs, T* __restrict__ u, const int* __restrict__ done)
{
    if (done && *done) return;
    const int n = mx * my * mz;
    for (int row = threadIdx.x; row < n; row += blockDim.x) {
        double s = 0.0;
        for (int col = 0; col < n; ++col) {
            const int ci = col % mx, cj = (col / mx) % my, ck = col / (mx * my);
            s += (double)ainv[(long long)row * n + col] * (double)rhs[(ci + 1) + (long long)sx * (cj + 1) + sp * (ck + k0)];
        }
        const int i = row % mx, j = (row / mx) % my, k = row / (mx * my);
        u[(i + 1) + (long long)sx * (j + 1) + sp * (k + k0)] = (T)s;
    }
}

// Partial sums of (rhs - L u)^2 over interior nodes, one per block, accumulated in fp64 (C10).
template <typename T, bool D3>
__global__ void __launch_bounds__(256) k_resnorm_partial_ref(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs,
                                                              double* __restrict__ partial, const int* __restrict__ done)
{
    if (done && *done) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = D3 ? (int)blockIdx.z + 1 : 0;
    double v = 0.0;
    if (i < p.sx && j < p.sy && i != 0 && j != 0) {
        const long long c = i + (long long)p.sx * j + p.sp * k;
        const T f = rhs ? rhs[c] : T(0);
        const double r = (double)(f - apply_L<T, D3>(p, u, c, k));
        v = r * r;
    }
    v = block_sum<256>(v);
    if (threadIdx.x == 0 && threadIdx.y == 0)
        partial[blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = v;
}

// Deterministic final reduction + stop rule (C10; stop_rule in mhs_device.cuh): one block, fixed summation order.
__global__ void __launch_bounds__(1024) k_norm_final(const double* __restrict__ partial, long long n, Ctl* ctl, int mode)
{
    pdl_enter();
    if (mode == 1 && ctl->done) return;
    double v = 0.0;
    for (long long q = threadIdx.x; q < n; q += 1024) v += partial[q];
    v = block_sum<1024>(v);
    if (threadIdx.x == 0) stop_rule(ctl, sqrt(v), mode);
}

// dense (nx,ny,nz) -> internal layout.  Walls (i = 0, j = 0, top plane, and the bottom plane unless
// keep_bottom) are written as zeros.
template <typename T>
__global__ void __launch_bounds__(256) k_pack(int nx, int ny, int nz, int sx, int sy, long long sp, const T* __restrict__ dense,
                                               T* __restrict__ dst, int keep_bottom, int negate, int is3d)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= sx || j >= sy) return;
    T v = T(0);
    const bool wall = (i == 0 || j == 0 || (is3d && (k == nz - 1 || (k == 0 && !keep_bottom))));
    if (!wall) {
        v = dense[i + (long long)nx * (j + (long long)ny * k)];
        if (negate) v = -v;
    }
    dst[i + (long long)sx * j + sp * k] = v;
}

// internal -> dense (all nx*ny*nz nodes; the aliased layout returns the wall zeros by itself).
template <typename T>
__global__ void __launch_bounds__(256) k_unpack(int nx, int ny, int sx, long long sp, const T* __restrict__ src, T* __restrict__ dense)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= nx || j >= ny) return;
    dense[i + (long long)nx * (j + (long long)ny * k)] = src[i + (long long)sx * j + sp * k];
}

// ------------------------------------------------------------------------------------------------
// Field recovery, reference version: one thread per node evaluates everything from P directly
// (eqs 9-10; C13-C15).  ft = xi[nz] | dxi[nz] | p_b[nz] | rho_b[nz].
// ------------------------------------------------------------------------------------------------
template <typename T>
struct FieldsP {
    int nx, ny, nz, sx;
    long long sp;
    T alpha, i2hx, i2hy, i2hz, ihx2, ihy2, i2mu0, imu0, ig;
    const T* ft;
};

template <typename T>
__device__ __forceinline__ bool is_wall(const FieldsP<T>& q, int i, int j, int k)
{
    return i <= 0 || j <= 0 || i >= q.nx - 1 || j >= q.ny - 1 || k >= q.nz - 1;
}
template <typename T>
__device__ __forceinline__ T Pat(const FieldsP<T>& q, const T* P, int i, int j, int k)
{
    return P[i + (long long)q.sx * j + q.sp * k];
}
template <typename T>
__device__ __forceinline__ T dzP(const FieldsP<T>& q, const T* P, int i, int j, int k)
{
    if (k == 0) return (T(-3) * Pat(q, P, i, j, 0) + T(4) * Pat(q, P, i, j, 1) - Pat(q, P, i, j, 2)) * q.i2hz;
    return (Pat(q, P, i, j, k + 1) - Pat(q, P, i, j, k - 1)) * q.i2hz;
}
template <typename T>
__device__ __forceinline__ T Bz_at(const FieldsP<T>& q, const T* P, int i, int j, int k)
{
    if (is_wall(q, i, j, k)) return T(0);
    const T uc = Pat(q, P, i, j, k);
    const T dxx = (Pat(q, P, i + 1, j, k) - T(2) * uc + Pat(q, P, i - 1, j, k)) * q.ihx2;
    const T dyy = (Pat(q, P, i, j + 1, k) - T(2) * uc + Pat(q, P, i, j - 1, k)) * q.ihy2;
    return -(dxx + dyy);
}

template <typename T>
__global__ void __launch_bounds__(256) k_fields_ref(FieldsP<T> q, const T* __restrict__ P, T* __restrict__ Bx, T* __restrict__ By,
                                                     T* __restrict__ Bz, T* __restrict__ pp, T* __restrict__ rho, int kstride)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * kstride;
    if (i >= q.nx || j >= q.ny) return;
    const long long d = i + (long long)q.nx * (j + (long long)q.ny * k);
    const T xi = q.ft[k], dxi = q.ft[q.nz + k], pb = q.ft[2 * q.nz + k], rb = q.ft[3 * q.nz + k];
    T bx = T(0), by = T(0), bz = T(0), pv = pb, rv = rb;
    if (!is_wall(q, i, j, k)) {
        bz = Bz_at(q, P, i, j, k);
        bx = q.alpha * (Pat(q, P, i, j + 1, k) - Pat(q, P, i, j - 1, k)) * q.i2hy + (dzP(q, P, i + 1, j, k) - dzP(q, P, i - 1, j, k)) * q.i2hx;
        by = -q.alpha * (Pat(q, P, i + 1, j, k) - Pat(q, P, i - 1, j, k)) * q.i2hx + (dzP(q, P, i, j + 1, k) - dzP(q, P, i, j - 1, k)) * q.i2hy;
        if (pp || rho) {
            const T dxBz = (Bz_at(q, P, i + 1, j, k) - Bz_at(q, P, i - 1, j, k)) * q.i2hx;
            const T dyBz = (Bz_at(q, P, i, j + 1, k) - Bz_at(q, P, i, j - 1, k)) * q.i2hy;
            T dzBz;
            if (k == 0) dzBz = (T(-3) * bz + T(4) * Bz_at(q, P, i, j, 1) - Bz_at(q, P, i, j, 2)) * q.i2hz;
            else dzBz = (Bz_at(q, P, i, j, k + 1) - Bz_at(q, P, i, j, k - 1)) * q.i2hz;
            pv = pb - xi * bz * bz * q.i2mu0;
            rv = rb + q.ig * (dxi * bz * bz * q.i2mu0 + q.imu0 * xi * (bx * dxBz + by * dyBz + bz * dzBz));
        }
    }
    if (Bx) { Bx[d] = bx; By[d] = by; Bz[d] = bz; }
    if (pp) pp[d] = pv;
    if (rho) rho[d] = rv;
}

// ------------------------------------------------------------------------------------------------
// host-side launchers (dtype / dimension dispatch)
// ------------------------------------------------------------------------------------------------
template <typename T>
static LP<T> make_lp(const mhs_ctx* c, const Level& lv)
{
    LP<T> p;
    p.nx = lv.nx; p.ny = lv.ny; p.nz = lv.nz; p.sx = lv.sx; p.sy = lv.sy; p.sp = lv.sp;
    p.tab = (const T*)lv.tab;
    p.cz = lv.dim == 3 ? (T)(1.0 / (lv.hz * lv.hz)) : T(0);
    p.a2 = lv.dim == 3 ? (T)(c->alpha * c->alpha) : T(0);
    return p;
}

static inline dim3 grid_xyk(const Level& lv, dim3 b)
{
    return dim3((lv.sx + b.x - 1) / b.x, (lv.sy + b.y - 1) / b.y, lv.dim == 3 ? lv.nz - 2 : 1);
}

#define DISPATCH(c, lv, EXPR_T_D3)                                      \
    do {                                                                \
        if ((c)->es == 8) {                                             \
            typedef double T;                                           \
            if ((lv).dim == 3) { constexpr bool D3 = true; EXPR_T_D3; } \
            else { constexpr bool D3 = false; EXPR_T_D3; }              \
        } else {                                                        \
            typedef float T;                                            \
            if ((lv).dim == 3) { constexpr bool D3 = true; EXPR_T_D3; } \
            else { constexpr bool D3 = false; EXPR_T_D3; }              \
        }                                                               \
    } while (0)

void launch_smooth_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done)
{
    const dim3 b(32, 8);
    count_launch(c);
    DISPATCH(c, lv, (k_smooth_ref<T, D3><<<grid_xyk(lv, b), b, 0, c->stream>>>(make_lp<T>(c, lv), (const T*)u, (const T*)rhs, (T*)out, done)));
}

void launch_residual_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* r, const int* done)
{
    const dim3 b(32, 8);
    count_launch(c);
    DISPATCH(c, lv, (k_residual_ref<T, D3><<<grid_xyk(lv, b), b, 0, c->stream>>>(make_lp<T>(c, lv), (const T*)u, (const T*)rhs, (T*)r, done)));
}

void launch_restrict_ref(mhs_ctx* c, const Level& f, const void* r, const Level& co, void* rhs_c, const int* done)
{
    const dim3 b(32, 8);
    count_launch(c);
    DISPATCH(c, co, (k_restrict_ref<T, D3><<<grid_xyk(co, b), b, 0, c->stream>>>(f.sx, f.sp, (const T*)r, co.sx, co.sy, co.sp, (T*)rhs_c, done)));
}

void launch_prolong_ref(mhs_ctx* c, const Level& f, void* u, const Level& co, const void* ec, const int* done)
{
    const dim3 b(32, 8);
    count_launch(c);
    DISPATCH(c, f, (k_prolong_ref<T, D3><<<grid_xyk(f, b), b, 0, c->stream>>>(f.sx, f.sy, f.sp, (T*)u, co.sx, co.sp, (const T*)ec, done)));
}

void launch_coarse_solve(mhs_ctx* c, const Level& lv, void* u, const void* rhs, const int* done)
{
    const int mx = lv.nx - 2, my = lv.ny - 2, mz = lv.dim == 3 ? lv.nz - 2 : 1, k0 = lv.dim == 3 ? 1 : 0;
    count_launch(c);
    if (c->es == 8)
        k_coarse_solve<double><<<1, 256, 0, c->stream>>>(mx, my, mz, lv.sx, lv.sp, k0, (const double*)lv.ainv, (const double*)rhs, (double*)u, done);
    else
        k_coarse_solve<float><<<1, 256, 0, c->stream>>>(mx, my, mz, lv.sx, lv.sp, k0, (const float*)lv.ainv, (const float*)rhs, (float*)u, done);
}

long long launch_resnorm_partial_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, const int* done)
{
    const dim3 b(32, 8);
    const dim3 g = grid_xyk(lv, b);
    count_launch(c);
    DISPATCH(c, lv, (k_resnorm_partial_ref<T, D3><<<g, b, 0, c->stream>>>(make_lp<T>(c, lv), (const T*)u, (const T*)rhs, c->partial, done)));
    return (long long)g.x * g.y * g.z;
}

long long resnorm_partial_capacity(const Level& lv)
{
    const dim3 b(32, 8);
    const dim3 g = grid_xyk(lv, b);
    return (long long)g.x * g.y * g.z;
}

void launch_norm_final(mhs_ctx* c, long long n, int mode)
{
    count_launch(c);
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_norm_final); return 1; });
    launch_pdl(c, k_norm_final, dim3(1), dim3(1024), 0, (const double*)c->partial, n, c->ctl, mode);
}

void launch_pack(mhs_ctx* c, const Level& lv, const void* dense, void* dst, bool keep_bottom, bool negate)
{
    const dim3 b(32, 8);
    const dim3 g((lv.sx + 31) / 32, (lv.sy + 7) / 8, lv.nz);
    count_launch(c);
    if (c->es == 8)
        k_pack<double><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, lv.sx, lv.sy, lv.sp, (const double*)dense, (double*)dst, keep_bottom, negate, lv.dim == 3);
    else
        k_pack<float><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, lv.sx, lv.sy, lv.sp, (const float*)dense, (float*)dst, keep_bottom, negate, lv.dim == 3);
}

void launch_unpack(mhs_ctx* c, const Level& lv, const void* src, void* dense)
{
    const dim3 b(32, 8);
    const dim3 g((lv.nx + 31) / 32, (lv.ny + 7) / 8, lv.nz);
    count_launch(c);
    if (c->es == 8)
        k_unpack<double><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.sx, lv.sp, (const double*)src, (double*)dense);
    else
        k_unpack<float><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.sx, lv.sp, (const float*)src, (float*)dense);
}

template <typename T>
static void fields_ref_t(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho, bool ends_only, bool dense)
{
    FieldsP<T> q;
    q.nx = lv.nx; q.ny = lv.ny; q.nz = lv.nz; q.sx = lv.sx; q.sp = lv.sp;
    if (dense) { q.sx = lv.nx; q.sp = (long long)lv.nx * lv.ny; }
    q.alpha = (T)c->alpha;
    q.i2hx = (T)(1.0 / (2.0 * lv.hx)); q.i2hy = (T)(1.0 / (2.0 * lv.hy)); q.i2hz = (T)(1.0 / (2.0 * lv.hz));
    q.ihx2 = (T)(1.0 / (lv.hx * lv.hx)); q.ihy2 = (T)(1.0 / (lv.hy * lv.hy));
    q.i2mu0 = (T)(1.0 / (2.0 * c->opt.mu0)); q.imu0 = (T)(1.0 / c->opt.mu0); q.ig = (T)(1.0 / c->opt.g);
    q.ft = (const T*)c->prof_tab;
    const dim3 b(32, 8);
    const dim3 g((lv.nx + 31) / 32, (lv.ny + 7) / 8, ends_only ? 2 : lv.nz);
    const long long N = lv.npts();
    T* Bx = (T*)B;
    k_fields_ref<T><<<g, b, 0, c->stream>>>(q, (const T*)P, Bx, Bx ? Bx + N : nullptr, Bx ? Bx + 2 * N : nullptr, (T*)p, (T*)rho,
                                            ends_only ? lv.nz - 1 : 1);
}

// ends_only: just the planes k = 0 and k = nz-1 (the rest is done by launch_fields_z)
void launch_fields_ref(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho, bool ends_only, bool dense)
{
    count_launch(c);
    if (c->es == 8) fields_ref_t<double>(c, lv, P, B, p, rho, ends_only, dense);
    else fields_ref_t<float>(c, lv, P, B, p, rho, ends_only, dense);
}

}  // namespace mhs
