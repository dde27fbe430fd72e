// Kernels of the solver variants of libmhs_b200 ("multigrid methods"; readings C25, C26):
//   * weighted z-LINE Jacobi relaxation: the smoother for strong (1 - xi) anisotropy -- the paper's xi_2 profile takes
//     1 - xi down to 0.05 near the base, where the vertical coupling of eq (8) is 20 times the horizontal one
//     and point relaxation stops smoothing;
//   * the two small kernels of the full-multigrid start: injection of the bottom-plane data to a coarse level and the
//     right-hand side the bottom data make for the exact coarsest solve.
#include "mhs_device.cuh"

namespace mhs {

// ------------------------------------------------------------------------------------------------
// out = u + omega d,   T d = rhs - L u on every z-line (i, j),   T = diag(L) + the two z-neighbours   (C25).
// T is the same tridiagonal matrix for every line, so its Thomas factors are per-plane constants computed once at create
// (zl = cp[nz] | 1/den[nz], den_k = D_k - a cp_{k-1}, cp_k = a / den_k, a = 1/hz^2).  One thread owns V adjacent lines
// (one 128-bit vector) and walks UP forming the residual and the forward elimination dp_k = (r_k - a dp_{k-1}) / den_k,
// which it parks in `out`; then DOWN with the back substitution d_k = dp_k - cp_k d_{k+1}, replacing dp_k by u_k + omega d_k.
// x-contiguous 128-bit accesses; a line's values are loaded once going up (its z-neighbours come from registers, its four
// horizontal neighbours from L1/L2) and once going down.  Traffic: read u twice, rhs once, dp once, write out twice.
// ------------------------------------------------------------------------------------------------
template <typename T> struct VV;
template <> struct VV<double> { static constexpr int N = 2; };
template <> struct VV<float> { static constexpr int N = 4; };
template <typename T> struct __align__(16) VecV { T v[VV<T>::N]; };
template <typename T> __device__ __forceinline__ VecV<T> ldvv(const T* p) { return *reinterpret_cast<const VecV<T>*>(p); }
template <typename T> __device__ __forceinline__ void stvv(T* p, const VecV<T>& a) { *reinterpret_cast<VecV<T>*>(p) = a; }

template <typename T, bool HAS_RHS>
__global__ void __launch_bounds__(128) k_zline(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, T* __restrict__ out,
                                                const T* __restrict__ zl, T omega, const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int V = VV<T>::N;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nv = p.sp / V;
    if (q >= nv) return;
    const long long c0 = q * V;                 // flat in-plane index of element 0
    const int i0 = (int)(c0 % p.sx), j = (int)(c0 / p.sx);
    if (j == 0) return;                          // wall row
    const T a = p.cz;
    const T* cp = zl;
    const T* iden = zl + p.nz;
    VecV<T> dn = ldvv(u + c0), cc = ldvv(u + c0 + p.sp), dp;
#pragma unroll
    for (int e = 0; e < V; ++e) dp.v[e] = T(0);
    for (int k = 1; k <= p.nz - 2; ++k) {
        const T* pl = u + c0 + p.sp * k;
        const VecV<T> up = ldvv(pl + p.sp), n = ldvv(pl + p.sx), s = ldvv(pl - p.sx);
        const T w = pl[-1], ea = pl[V];
        const T cx = p.tab[k], cy = p.tab[p.nz + k], id = iden[k];
        VecV<T> f;
        if (HAS_RHS) f = ldvv(rhs + c0 + p.sp * k);
#pragma unroll
        for (int e = 0; e < V; ++e) {
            const T ww = e == 0 ? w : cc.v[e - 1], ee = e == V - 1 ? ea : cc.v[e + 1];
            T lu = cx * lap1<T>(ee, ww, cc.v[e]) + cy * lap1<T>(n.v[e], s.v[e], cc.v[e]);
            lu += a * lap1<T>(up.v[e], dn.v[e], cc.v[e]) + p.a2 * cc.v[e];
            const T r = (HAS_RHS ? f.v[e] : T(0)) - lu;
            dp.v[e] = (r - a * dp.v[e]) * id;
        }
        stvv(out + c0 + p.sp * k, dp);
        dn = cc; cc = up;
    }
    // back substitution; element 0 of the first vector of a row is the wall column: it keeps its (zero) value
    VecV<T> d;
#pragma unroll
    for (int e = 0; e < V; ++e) d.v[e] = T(0);
    for (int k = p.nz - 2; k >= 1; --k) {
        const VecV<T> y = ldvv(out + c0 + p.sp * k), uc = ldvv(u + c0 + p.sp * k);
        const T ck = cp[k];
        VecV<T> o;
#pragma unroll
        for (int e = 0; e < V; ++e) {
            d.v[e] = y.v[e] - ck * d.v[e];
            o.v[e] = (i0 + e == 0) ? uc.v[e] : uc.v[e] + omega * d.v[e];
        }
        stvv(out + c0 + p.sp * k, o);
    }
}

template <typename T>
static LP<T> lp_make(const mhs_ctx* c, const Level& lv)
{
    LP<T> p;
    p.nx = lv.nx; p.ny = lv.ny; p.nz = lv.nz; p.sx = lv.sx; p.sy = lv.sy; p.sp = lv.sp;
    p.tab = (const T*)lv.tab;
    p.cz = (T)(1.0 / (lv.hz * lv.hz));
    p.a2 = (T)(c->alpha * c->alpha);
    return p;
}

bool zline_ok(const mhs_ctx* c, const Level& lv)
{
    const int V = c->es == 8 ? 2 : 4;
    return lv.dim == 3 && !lv.coarsest && lv.zl != nullptr && lv.sx % V == 0 && lv.nz >= 3;
}

void launch_zline(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done)
{
    count_launch(c);
    const int V = c->es == 8 ? 2 : 4;
    const unsigned nb = (unsigned)((lv.sp / V + 127) / 128);
#define ZL(T)                                                                                                               \
    do {                                                                                                                    \
        static PerDevice once;                                                                                              \
        per_device(once, c, [&] { prefer_l1(k_zline<T, true>); prefer_l1(k_zline<T, false>); return 1; });                  \
        if (rhs) launch_pdl(c, k_zline<T, true>, dim3(nb), dim3(128), 0, lp_make<T>(c, lv), (const T*)u, (const T*)rhs, (T*)out, \
                            (const T*)lv.zl, (T)c->opt.omega, done);                                                        \
        else launch_pdl(c, k_zline<T, false>, dim3(nb), dim3(128), 0, lp_make<T>(c, lv), (const T*)u, (const T*)rhs, (T*)out, \
                        (const T*)lv.zl, (T)c->opt.omega, done);                                                            \
    } while (0)
    if (c->es == 8) ZL(double);
    else ZL(float);
#undef ZL
}

// ------------------------------------------------------------------------------------------------
// Full-multigrid start (C26).  k_inject_bottom: bottom plane of a coarse level <- the finest level's bottom plane at
// every `stride`-th node (both in the aliased layout).  k_bottom_rhs: the right-hand side the bottom data b make for the
// interior unknowns of plane 1, rhs(i,j,1) = -b(i,j)/hz^2 (the exact coarsest solve applies A^-1 to it).
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_inject_bottom(int csx, int csy, const T* __restrict__ fine, int fsx, int stride, T* __restrict__ a,
                                                        T* __restrict__ b)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y;
    if (I >= csx || J >= csy) return;
    const T v = (I == 0 || J == 0) ? T(0) : fine[(long long)stride * I + (long long)fsx * stride * J];
    a[I + (long long)csx * J] = v;
    if (b) b[I + (long long)csx * J] = v;
}

template <typename T>
__global__ void __launch_bounds__(256) k_bottom_rhs(int sx, int sy, long long sp, T cz, const T* __restrict__ u, T* __restrict__ rhs)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= sx || j >= sy) return;
    rhs[i + (long long)sx * j + sp] = (i == 0 || j == 0) ? T(0) : -cz * u[i + (long long)sx * j];
}

void launch_inject_bottom(mhs_ctx* c, const Level& fine, const void* fine_u, const Level& lv, int stride, void* a, void* b)
{
    count_launch(c);
    const dim3 g((lv.sx + 255) / 256, lv.sy);
    if (c->es == 8) k_inject_bottom<double><<<g, 256, 0, c->stream>>>(lv.sx, lv.sy, (const double*)fine_u, fine.sx, stride, (double*)a, (double*)b);
    else k_inject_bottom<float><<<g, 256, 0, c->stream>>>(lv.sx, lv.sy, (const float*)fine_u, fine.sx, stride, (float*)a, (float*)b);
}

void launch_bottom_rhs(mhs_ctx* c, const Level& lv, const void* u, void* rhs)
{
    count_launch(c);
    const dim3 g((lv.sx + 255) / 256, lv.sy);
    const double cz = 1.0 / (lv.hz * lv.hz);
    if (c->es == 8) k_bottom_rhs<double><<<g, 256, 0, c->stream>>>(lv.sx, lv.sy, lv.sp, cz, (const double*)u, (double*)rhs);
    else k_bottom_rhs<float><<<g, 256, 0, c->stream>>>(lv.sx, lv.sy, lv.sp, (float)cz, (const float*)u, (float*)rhs);
}

}  // namespace mhs
