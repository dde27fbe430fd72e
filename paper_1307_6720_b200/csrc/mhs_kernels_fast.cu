// Tuned 3D kernels of libmhs_b200 for sm_100a (HBM-bound 7-point stencils; no tensor cores: nothing
// here is a dense contraction).  Common scheme ("flat z-streaming"):
//
//   * The aliased Dirichlet layout (mhs_internal.h) makes every plane one FLAT array: the x-neighbours
//     of an element are flat-1 / flat+1 even across row ends (what sits there is a wall zero), the
//     y-neighbours are flat-+sx.  A thread owns R vertically adjacent 128-bit vectors (double2 / float4)
//     and walks up in z keeping the planes k-1, k, k+1 of its R vectors in registers, so each element of
//     the iterate is loaded once per kernel by its owner (+ the two halo rows of the R-row strip, which
//     hit L1/L2) and z-neighbours never touch memory.
//   * x-neighbours across vectors come from warp shuffles; only lanes 0 and 31 issue a scalar load.
//   * c_k/hx^2, c_k/hy^2, omega/D_k are per-plane scalars from a small table (L1-resident).
//   * The residual rhs - L u of the INPUT iterate is an intermediate of the Jacobi update, so its squared
//     norm is accumulated for free (warp shuffles + one partial per block): the stop test needs no pass of
//     its own.
//   * Grids are sized to fill a whole number of waves on the 148 SMs (z-chunk length is the free parameter);
//     consecutive kernels traverse the z-chunks in opposite order so that the tail of what the previous
//     kernel wrote is still in the 126 MB L2 when the next one starts.
#include <cstdlib>

#include "mhs_device.cuh"

namespace mhs {

template <typename T> struct VN;
template <> struct VN<double> { static constexpr int N = 2; };
template <> struct VN<float> { static constexpr int N = 4; };

template <typename T>
struct __align__(16) Vec {
    T v[VN<T>::N];
};

template <typename T>
__device__ __forceinline__ Vec<T> ldv(const T* p) { return *reinterpret_cast<const Vec<T>*>(p); }
template <typename T>
__device__ __forceinline__ void stv(T* p, const Vec<T>& a) { *reinterpret_cast<Vec<T>*>(p) = a; }

__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_up1(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_dn1(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// rhs - L u for the V elements of one vector.  cw/ce: the elements left / right of the vector.
template <typename T>
__device__ __forceinline__ void residual_vec(const Vec<T>& c, T cw, T ce, const Vec<T>& n, const Vec<T>& s, const Vec<T>& up,
                                             const Vec<T>& dn, const Vec<T>* f, T cx, T cy, T cz, T a2, Vec<T>& r)
{
    constexpr int V = VN<T>::N;
#pragma unroll
    for (int e = 0; e < V; ++e) {
        const T w = e == 0 ? cw : c.v[e - 1];
        const T ea = e == V - 1 ? ce : c.v[e + 1];
        T lu = cx * lap1<T>(ea, w, c.v[e]) + cy * lap1<T>(n.v[e], s.v[e], c.v[e]);
        lu += cz * lap1<T>(up.v[e], dn.v[e], c.v[e]) + a2 * c.v[e];
        r.v[e] = (f ? f->v[e] : T(0)) - lu;
    }
}

// ------------------------------------------------------------------------------------------------
// One weighted-Jacobi sweep (a2) over the z-chunk of this block.
//   STORE : write out = u + (omega/D_k) r          NORM : accumulate sum r^2 into partial[block]
// Work item q <-> (row group g, x vector xv): rows j0 = g*R .. j0+R-1, elements i0 = xv*V .. i0+V-1.
// ------------------------------------------------------------------------------------------------
//   ZERO2 : the iterate is the result of the first sweep from the zero initial guess of a coarse-grid correction,
//           u1 = (omega/D_k) rhs (0 on the planes k = 0, nz-1 and on the walls, where rhs is 0); it is never stored:
//           `u` is not read, its values are formed from rhs on the fly, so "two sweeps from zero" is ONE pass that
//           reads rhs and writes u2.
template <typename T, int R, bool HAS_RHS, bool STORE, bool NORM, bool ZERO2>
__global__ void __launch_bounds__(128) k_smooth_z(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, T* __restrict__ out,
                                                   int kchunk, int nzc, int reverse, double* __restrict__ partial,
                                                   const int* __restrict__ done)
{
    static_assert(!ZERO2 || (HAS_RHS && STORE && !NORM), "ZERO2 is a plain sweep with a right-hand side");
    pdl_enter();
    if (done && *done) return;
    if (ZERO2) u = rhs;
    constexpr int V = VN<T>::N;
    const int nvx = p.sx / V;
    const int ngroups = (p.sy + R - 1) / R;
    const long long total = (long long)ngroups * nvx;
    const long long q0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = q0 < total;
    const long long q = active ? q0 : 0;   // idle lanes shadow item 0: its first element is a wall zero, which
                                           // is exactly the right-hand neighbour the last active lane needs
    const int g = (int)(q / nvx), xv = (int)(q - (long long)g * nvx);
    const int i0 = xv * V, j0 = g * R;
    const int lane = threadIdx.x & 31;
    const int zc = reverse ? nzc - 1 - (int)blockIdx.y : (int)blockIdx.y;
    const int kb = 1 + zc * kchunk;
    const int ke = min(kb + kchunk, p.nz - 1);
    const long long base = i0 + (long long)p.sx * j0;
    const T* tab = p.tab;

    const T* wz = tab + 9 * (long long)p.nz;   // omega/D_k on interior planes, 0 on k = 0 and k = nz-1
    Vec<T> cm[R], cc[R], cp[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        cm[r] = ldv(u + base + (long long)p.sx * r + p.sp * (kb - 1));
        cc[r] = ldv(u + base + (long long)p.sx * r + p.sp * kb);
        if (ZERO2) {
            const T a = wz[kb - 1], b = wz[kb];
#pragma unroll
            for (int e = 0; e < V; ++e) { cm[r].v[e] *= a; cc[r].v[e] *= b; }
        }
    }
    double acc = 0.0;
    for (int k = kb; k < ke; ++k) {
        const T* pl = u + base + p.sp * k;
#pragma unroll
        for (int r = 0; r < R; ++r) cp[r] = ldv(pl + p.sp + (long long)p.sx * r);
        Vec<T> ntop = ldv(pl + (long long)p.sx * R);
        Vec<T> sbot = ldv(pl - p.sx);
        const T cx = tab[k], cy = tab[p.nz + k], wk = tab[3 * p.nz + k];
        if (ZERO2) {
            const T a = wz[k + 1];
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int e = 0; e < V; ++e) cp[r].v[e] *= a;
#pragma unroll
            for (int e = 0; e < V; ++e) { ntop.v[e] *= wk; sbot.v[e] *= wk; }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            T cw = shfl_up1(cc[r].v[V - 1]);
            T ce = shfl_dn1(cc[r].v[0]);
            if (lane == 0) cw = ZERO2 ? wk * pl[(long long)p.sx * r - 1] : pl[(long long)p.sx * r - 1];
            if (lane == 31) ce = ZERO2 ? wk * pl[(long long)p.sx * r + V] : pl[(long long)p.sx * r + V];
            Vec<T> f, res;
            if (HAS_RHS) f = ldv(rhs + base + p.sp * k + (long long)p.sx * r);
            residual_vec<T>(cc[r], cw, ce, r == R - 1 ? ntop : cc[r + 1 < R ? r + 1 : r], r == 0 ? sbot : cc[r > 0 ? r - 1 : 0],
                            cp[r], cm[r], HAS_RHS ? &f : nullptr, cx, cy, p.cz, p.a2, res);
            const bool rowok = active && (j0 + r < p.sy) && (j0 + r > 0);
            Vec<T> o;
#pragma unroll
            for (int e = 0; e < V; ++e) {
                const bool wall = (i0 + e == 0);
                o.v[e] = wall ? cc[r].v[e] : cc[r].v[e] + wk * res.v[e];
                if (NORM && rowok && !wall) acc += (double)res.v[e] * (double)res.v[e];
            }
            if (STORE && rowok) stv(out + base + p.sp * k + (long long)p.sx * r, o);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) { cm[r] = cc[r]; cc[r] = cp[r]; }
    }
    if (NORM) {
        acc = block_sum<128>(acc);
        if (threadIdx.x == 0) partial[blockIdx.x + (long long)gridDim.x * blockIdx.y] = acc;
    }
}

// u = (omega/D_k) rhs : the first sweep from the zero initial guess of a coarse-grid correction
// (u + w (rhs - L 0) with u = 0), saving the zero fill and one read of u.
template <typename T>
__global__ void __launch_bounds__(256) k_scale_rhs(LP<T> p, const T* __restrict__ rhs, T* __restrict__ u, const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int V = VN<T>::N;
    const long long nv = p.sp / V;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int k = blockIdx.y + 1;
    if (q >= nv) return;
    const T wk = p.tab[3 * p.nz + k];
    Vec<T> f = ldv(rhs + q * V + p.sp * k);
#pragma unroll
    for (int e = 0; e < V; ++e) f.v[e] *= wk;
    stv(u + q * V + p.sp * k, f);
}

// ------------------------------------------------------------------------------------------------
// Residual + full-weighting restriction fused (a3 + a4): rhs_c = R (rhs - L u), never storing r.
// A thread owns rows j0-1 .. j0+R-1 (R even, j0 even) of one x vector: the residuals of R+1 rows give the
// R/2 coarse rows j0/2 .. ; the x part of the weighting takes the odd left neighbour from the lane below
// (warps overlap by one vector: lane 0 only feeds lane 1), the z part is accumulated while streaming:
// odd fine planes close one coarse plane with weight 1/4 and open the next.
// ------------------------------------------------------------------------------------------------
template <typename T, int R, bool HAS_RHS>
__global__ void __launch_bounds__(128) k_resid_restrict_z(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, int csx,
                                                           long long csp, int cnz, T* __restrict__ rc, int Kchunk, int nzc, int reverse,
                                                           const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int V = VN<T>::N;
    constexpr int VC = V / 2;
    constexpr int RR = R + 1;
    const int nvx = p.sx / V;
    const int ngroups = (p.sy + R - 1) / R;
    const long long total = (long long)ngroups * nvx;
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long q0 = warp * 31 + lane - 1;
    const bool active = q0 >= 0 && q0 < total && lane > 0;
    const long long q = (q0 >= 0 && q0 < total) ? q0 : 0;
    const int g = (int)(q / nvx), xv = (int)(q - (long long)g * nvx);
    const int i0 = xv * V, j0 = g * R;
    const int zc = reverse ? nzc - 1 - (int)blockIdx.y : (int)blockIdx.y;
    const int Kb = 1 + zc * Kchunk;
    const int Ke = min(Kb + Kchunk, cnz - 1);
    if (Kb >= Ke) return;
    const long long base = i0 + (long long)p.sx * (j0 - 1);   // row t = 0 is fine row j0-1
    const T* tab = p.tab;

    Vec<T> cm[RR], cc[RR], cp[RR];
    const int k0 = 2 * Kb - 1;
#pragma unroll
    for (int t = 0; t < RR; ++t) {
        cm[t] = ldv(u + base + (long long)p.sx * t + p.sp * (k0 - 1));
        cc[t] = ldv(u + base + (long long)p.sx * t + p.sp * k0);
    }
    T accA[R / 2][VC];
#pragma unroll
    for (int s = 0; s < R / 2; ++s)
#pragma unroll
        for (int m = 0; m < VC; ++m) accA[s][m] = T(0);

    for (int k = k0; k <= 2 * Ke - 1; ++k) {
        const T* pl = u + base + p.sp * k;
#pragma unroll
        for (int t = 0; t < RR; ++t) cp[t] = ldv(pl + p.sp + (long long)p.sx * t);
        const Vec<T> ntop = ldv(pl + (long long)p.sx * RR);
        const Vec<T> sbot = ldv(pl - p.sx);
        const T cx = tab[k], cy = tab[p.nz + k];
        T tx[RR][VC];
#pragma unroll
        for (int t = 0; t < RR; ++t) {
            T cw = shfl_up1(cc[t].v[V - 1]);
            T ce = shfl_dn1(cc[t].v[0]);
            if (lane == 0) cw = pl[(long long)p.sx * t - 1];
            if (lane == 31) ce = pl[(long long)p.sx * t + V];
            Vec<T> f, res;
            if (HAS_RHS) f = ldv(rhs + base + p.sp * k + (long long)p.sx * t);
            residual_vec<T>(cc[t], cw, ce, t == RR - 1 ? ntop : cc[t + 1 < RR ? t + 1 : t], t == 0 ? sbot : cc[t > 0 ? t - 1 : 0],
                            cp[t], cm[t], HAS_RHS ? &f : nullptr, cx, cy, p.cz, p.a2, res);
            const int j = j0 - 1 + t;
            const bool rowok = j > 0 && j < p.sy;   // wall rows (and the aliased rows beyond them) carry r = 0
#pragma unroll
            for (int e = 0; e < V; ++e)
                if (!rowok || (i0 + e == 0)) res.v[e] = T(0);
            // x weighting: coarse element m sits on fine element 2m of this vector
            const T left = shfl_up1(res.v[V - 1]);
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                const T l = m == 0 ? left : res.v[2 * m - 1];
                tx[t][m] = T(0.5) * res.v[2 * m] + T(0.25) * (l + res.v[2 * m + 1]);
            }
        }
        const bool odd = (k & 1) != 0;
#pragma unroll
        for (int s = 0; s < R / 2; ++s) {
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                const T ty = T(0.5) * tx[2 * s + 1][m] + T(0.25) * (tx[2 * s][m] + tx[2 * s + 2][m]);
                if (!odd) {
                    accA[s][m] += T(0.5) * ty;
                } else {
                    const T closed = accA[s][m] + T(0.25) * ty;
                    accA[s][m] = T(0.25) * ty;
                    if (k > k0) {
                        const int K = (k - 1) >> 1;
                        const int I = (i0 >> 1) + m, J = (j0 >> 1) + s;
                        if (active && I > 0 && J > 0 && (j0 + 2 * s) < p.sy)
                            rc[I + (long long)csx * J + csp * K] = closed;
                    }
                }
            }
        }
#pragma unroll
        for (int t = 0; t < RR; ++t) { cm[t] = cc[t]; cc[t] = cp[t]; }
    }
}

// ------------------------------------------------------------------------------------------------
// Trilinear prolongation + correction (a6): u += P e_c, one fine vector per thread.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_prolong_v(int sx, int sy, long long sp, T* __restrict__ u, int csx, long long csp,
                                                    const T* __restrict__ ec, int reverse, int nzi, const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int V = VN<T>::N;
    constexpr int VC = V / 2;
    const long long nv = sp / V;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int k = (reverse ? nzi - 1 - (int)blockIdx.y : (int)blockIdx.y) + 1;
    if (q >= nv) return;
    const long long flat = q * V;
    const int j = (int)(flat / sx), i0 = (int)(flat - (long long)j * sx);
    if (j == 0) return;
    const int I0 = i0 >> 1, J0 = j >> 1, J1 = (j + 1) >> 1, K0 = k >> 1, K1 = (k + 1) >> 1;
    // sum the four (J,K) corner rows first, then interpolate in x
    T c[VC + 1];
#pragma unroll
    for (int m = 0; m <= VC; ++m) {
        const long long o = I0 + m;
        c[m] = (ec[o + (long long)csx * J0 + csp * K0] + ec[o + (long long)csx * J1 + csp * K0]) +
               (ec[o + (long long)csx * J0 + csp * K1] + ec[o + (long long)csx * J1 + csp * K1]);
    }
    Vec<T> a = ldv(u + flat + sp * k);
#pragma unroll
    for (int e = 0; e < V; ++e) {
        const T s = (e & 1) ? (c[e >> 1] + c[(e >> 1) + 1]) : T(2) * c[e >> 1];
        if (i0 + e != 0) a.v[e] += T(0.125) * s;
    }
    stv(u + flat + sp * k, a);
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
template <typename T>
static LP<T> lp_of(const mhs_ctx* c, const Level& lv)
{
    LP<T> p;
    p.nx = lv.nx; p.ny = lv.ny; p.nz = lv.nz; p.sx = lv.sx; p.sy = lv.sy; p.sp = lv.sp;
    p.tab = (const T*)lv.tab;
    p.cz = (T)(1.0 / (lv.hz * lv.hz));
    p.a2 = (T)(c->alpha * c->alpha);
    return p;
}

bool fast_ok(const mhs_ctx* c, const Level& lv)
{
    const int V = c->es == 8 ? 2 : 4;
    return lv.dim == 3 && !lv.coarsest && lv.sx % V == 0 && lv.sx >= V && lv.nz >= 3;
}

// z-chunk length such that the grid is (just under) a whole number of waves of `slots` resident blocks.
static int pick_chunks(long long xy_blocks, int planes, int slots, int min_chunk)
{
    int best = 1;
    double best_score = -1.0;
    const int maxc = planes / min_chunk > 0 ? planes / min_chunk : 1;
    for (int nc = 1; nc <= maxc; ++nc) {
        const int len = (planes + nc - 1) / nc;
        const int real = (planes + len - 1) / len;
        const double blocks = (double)xy_blocks * real;
        const double waves = blocks / slots;
        const double eff = waves / std::ceil(waves);                  // last-wave quantisation
        const double halo = (double)len / (len + 2);                  // 2 redundant planes per chunk
        const double par = std::min(1.0, blocks / slots);             // enough blocks to fill the machine
        const double score = eff * halo * par;
        if (score > best_score + 1e-9) { best_score = score; best = real; }
    }
    return best;
}

// Levels that fit in the L2 several times over (<= ~5 M nodes: 129^3 and below) are not bandwidth problems but
// parallelism problems: they get one row per thread and short z-chunks, so that even 65^3 fills the 148 SMs.
bool mid_level(const mhs_ctx* c, const Level& lv) { return !(c->opt.flags & MHS_FLAG_BIG_LEVEL_KERNELS) && lv.npts() <= c->mid_pts; }

template <typename T, int R, bool HAS_RHS, bool STORE, bool NORM, bool ZERO2>
static long long smooth_z_t(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int reverse, const int* done)
{
    constexpr int V = VN<T>::N;
    auto kern = k_smooth_z<T, R, HAS_RHS, STORE, NORM, ZERO2>;
    static PerDevice slots_pd;
    const int slots = per_device(slots_pd, c, [&] {
        prefer_l1(kern);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 128, 0);
        return std::max(1, nb) * c->num_sms;
    });
    const long long items = (long long)((lv.sy + R - 1) / R) * (lv.sx / V);
    const long long xb = (items + 127) / 128;
    const int planes = lv.nz - 2;
    // L2-resident levels: parallelism first -- one plane per thread up to 65^3, two above (measured per level at 257^3:
    // 33^3 16.1 -> 13.8 us, 65^3 20.9 -> 17.5 us, 129^3 49.6 -> 45.4 us against the wave-filling heuristic)
    const int nzc = R == 1 ? (lv.npts() <= 300000LL ? planes : (planes + 1) / 2) : pick_chunks(xb, planes, slots, 8);
    const int kchunk = (planes + nzc - 1) / nzc;
    const int nzc2 = (planes + kchunk - 1) / kchunk;
    dim3 grid((unsigned)xb, (unsigned)nzc2);
    launch_pdl(c, kern, grid, dim3(128), 0, lp_of<T>(c, lv), (const T*)u, (const T*)rhs, (T*)out, kchunk, nzc2, reverse, c->partial, done);
    return xb * nzc2;
}

// mode: 0 = sweep, 1 = sweep + norm of the input residual, 2 = norm only, 3 = the first TWO sweeps from the zero
// initial guess (u is not read).  Returns the number of partials.
long long launch_smooth_z(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int mode, int reverse, const int* done)
{
    count_launch(c);
#define SZ(T, R)                                                                                                     \
    do {                                                                                                             \
        if (mode == 3) return smooth_z_t<T, R, true, true, false, true>(c, lv, u, rhs, out, reverse, done);          \
        if (rhs) {                                                                                                   \
            if (mode == 0) return smooth_z_t<T, R, true, true, false, false>(c, lv, u, rhs, out, reverse, done);     \
            if (mode == 1) return smooth_z_t<T, R, true, true, true, false>(c, lv, u, rhs, out, reverse, done);      \
            return smooth_z_t<T, R, true, false, true, false>(c, lv, u, rhs, out, reverse, done);                    \
        } else {                                                                                                     \
            if (mode == 0) return smooth_z_t<T, R, false, true, false, false>(c, lv, u, rhs, out, reverse, done);    \
            if (mode == 1) return smooth_z_t<T, R, false, true, true, false>(c, lv, u, rhs, out, reverse, done);     \
            return smooth_z_t<T, R, false, false, true, false>(c, lv, u, rhs, out, reverse, done);                   \
        }                                                                                                            \
    } while (0)
    const bool mid = mid_level(c, lv);
    if (c->es == 8) { if (mid) SZ(double, 1); SZ(double, 4); }
    else { if (mid) SZ(float, 1); SZ(float, 4); }
#undef SZ
    return 0;
}

long long smooth_z_partial_capacity(const mhs_ctx* c, const Level& lv)
{
    const int V = c->es == 8 ? 2 : 4;
    const int R = mid_level(c, lv) ? 1 : 4;
    const long long items = (long long)((lv.sy + R - 1) / R) * (lv.sx / V);
    return ((items + 127) / 128) * (long long)std::max(1, lv.nz - 2);   // (at most one z-chunk per plane)
}

// TWO Jacobi sweeps in one launch on the smallest grid-kernel level (33^3: up to c->s2_pts nodes), one thread per node: sweep 1 is
// formed on the fly at the seven nodes sweep 2 reads (a wall neighbour keeps its value).  Seven times the arithmetic of a
// sweep -- but on these levels a sweep kernel is ~4.5 us of launch and load latency whatever it computes, and the two
// post-smoothing sweeps of a level were two dependent launches.  Same expressions as one sweep after the other.
template <typename T>
__global__ void __launch_bounds__(128) k_smooth2_node(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, T* __restrict__ out,
                                                      const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    const int i = 1 + (int)(blockIdx.x * blockDim.x + threadIdx.x);
    const int j = 1 + (int)(blockIdx.y * blockDim.y + threadIdx.y);
    const int k = 1 + (int)blockIdx.z;
    if (i > p.nx - 2 || j > p.ny - 2) return;
    const long long c = i + (long long)p.sx * j + p.sp * k;
    auto sweep1 = [&](long long q, int kk, bool interior) -> T {
        if (!interior) return u[q];     // a wall node passes through (zero, or the bottom data of a full-multigrid level)
        return u[q] + p.tab[3 * p.nz + kk] * (rhs[q] - apply_L<T, true>(p, u, q, kk));
    };
    const T uc = sweep1(c, k, true);
    const T e = sweep1(c + 1, k, i + 1 <= p.nx - 2), w = sweep1(c - 1, k, i - 1 >= 1);
    const T n = sweep1(c + p.sx, k, j + 1 <= p.ny - 2), s = sweep1(c - p.sx, k, j - 1 >= 1);
    const T up = sweep1(c + p.sp, k + 1, k + 1 <= p.nz - 2), dn = sweep1(c - p.sp, k - 1, k - 1 >= 1);
    const T lu = p.tab[k] * lap1<T>(e, w, uc) + p.tab[p.nz + k] * lap1<T>(n, s, uc) + p.cz * lap1<T>(up, dn, uc) + p.a2 * uc;
    out[c] = uc + p.tab[3 * p.nz + k] * (rhs[c] - lu);
}

// Residual + full weighting on the smallest grid-kernel level as a "box" kernel: a CTA owns CT^3 coarse nodes, forms the
// residual at the (2 CT + 1)^3 fine nodes under them into shared memory (every one of them is an interior node) and
// weights it from there -- x, then y, then z, as everywhere else.  k_resid_restrict_z walks a z-column per thread; on a
// 33^3 level that is 45 CTAs and a chain of dependent plane loads (9.4 us against 3.9 us for a sweep of the same level).
template <typename T, int CT>
__global__ void __launch_bounds__(128) k_resid_restrict_box(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, int csx, long long csp,
                                                            int cnx, int cny, int cnz, T* __restrict__ rc, const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int F = 2 * CT + 1;
    __shared__ T r[F * F * F];
    const int I0 = 1 + CT * (int)blockIdx.x, J0 = 1 + CT * (int)blockIdx.y, K0 = 1 + CT * (int)blockIdx.z;   // first coarse node of the box
    const int fi0 = 2 * I0 - 1, fj0 = 2 * J0 - 1, fk0 = 2 * K0 - 1;                                           // first fine node under it
    for (int q = (int)threadIdx.x; q < F * F * F; q += (int)blockDim.x) {
        const int a = q % F, b = (q / F) % F, c = q / (F * F);
        const int i = fi0 + a, j = fj0 + b, k = fk0 + c;
        T v = T(0);
        if (i <= p.nx - 2 && j <= p.ny - 2 && k <= p.nz - 2) {
            const long long g = i + (long long)p.sx * j + p.sp * k;
            v = rhs[g] - apply_L<T, true>(p, u, g, k);
        }
        r[q] = v;
    }
    __syncthreads();
    for (int q = (int)threadIdx.x; q < CT * CT * CT; q += (int)blockDim.x) {
        const int a = q % CT, b = (q / CT) % CT, c = q / (CT * CT);
        const int I = I0 + a, J = J0 + b, K = K0 + c;
        if (I > cnx - 2 || J > cny - 2 || K > cnz - 2) continue;
        const T* r0 = r + (2 * a + 1) + F * (2 * b + 1) + F * F * (2 * c + 1);
        T s = T(0);
#pragma unroll
        for (int dc = -1; dc <= 1; ++dc) {
            T sp = T(0);
#pragma unroll
            for (int db = -1; db <= 1; ++db) {
                const T* row = r0 + F * db + F * F * dc;
                const T sxv = T(0.25) * (row[-1] + row[1]) + T(0.5) * row[0];
                sp += (db == 0 ? T(0.5) : T(0.25)) * sxv;
            }
            s += (dc == 0 ? T(0.5) : T(0.25)) * sp;
        }
        rc[I + (long long)csx * J + csp * K] = s;
    }
}

bool resid_restrict_box_ok(const mhs_ctx* c, const Level& f) { return f.dim == 3 && f.nz >= 5 && f.rhs && f.npts() <= c->rb_pts && fast_ok(c, f); }

void launch_resid_restrict_box(mhs_ctx* c, const Level& f, const void* u, const void* rhs, const Level& co, void* rc, const int* done)
{
    constexpr int CT = 2;
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_resid_restrict_box<double, CT>); prefer_l1(k_resid_restrict_box<float, CT>); return 1; });
    count_launch(c);
    const dim3 grid((unsigned)((co.nx - 2 + CT - 1) / CT), (unsigned)((co.ny - 2 + CT - 1) / CT), (unsigned)((co.nz - 2 + CT - 1) / CT));
    if (c->es == 8)
        launch_pdl(c, k_resid_restrict_box<double, CT>, grid, dim3(128), 0, lp_of<double>(c, f), (const double*)u, (const double*)rhs, co.sx, co.sp,
                   co.nx, co.ny, co.nz, (double*)rc, done);
    else
        launch_pdl(c, k_resid_restrict_box<float, CT>, grid, dim3(128), 0, lp_of<float>(c, f), (const float*)u, (const float*)rhs, co.sx, co.sp, co.nx,
                   co.ny, co.nz, (float*)rc, done);
}

bool smooth2_node_ok(const mhs_ctx* c, const Level& lv)
{
    return lv.dim == 3 && lv.nz >= 3 && lv.rhs && lv.npts() <= c->s2_pts && fast_ok(c, lv);
}

void launch_smooth2_node(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done)
{
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_smooth2_node<double>); prefer_l1(k_smooth2_node<float>); return 1; });
    count_launch(c);
    const dim3 block(32, 4), grid((unsigned)((lv.nx - 2 + 31) / 32), (unsigned)((lv.ny - 2 + 3) / 4), (unsigned)(lv.nz - 2));
    if (c->es == 8) launch_pdl(c, k_smooth2_node<double>, grid, block, 0, lp_of<double>(c, lv), (const double*)u, (const double*)rhs, (double*)out, done);
    else launch_pdl(c, k_smooth2_node<float>, grid, block, 0, lp_of<float>(c, lv), (const float*)u, (const float*)rhs, (float*)out, done);
}

void launch_scale_rhs(mhs_ctx* c, const Level& lv, const void* rhs, void* u, const int* done)
{
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_scale_rhs<double>); prefer_l1(k_scale_rhs<float>); return 1; });
    count_launch(c);
    const int V = c->es == 8 ? 2 : 4;
    dim3 grid((unsigned)((lv.sp / V + 255) / 256), (unsigned)(lv.nz - 2));
    if (c->es == 8) k_scale_rhs<double><<<grid, 256, 0, c->stream>>>(lp_of<double>(c, lv), (const double*)rhs, (double*)u, done);
    else k_scale_rhs<float><<<grid, 256, 0, c->stream>>>(lp_of<float>(c, lv), (const float*)rhs, (float*)u, done);
}

template <typename T, int R, bool HAS_RHS>
static void resid_restrict_t(mhs_ctx* c, const Level& f, const void* u, const void* rhs, const Level& co, void* rc, int reverse, const int* done)
{
    constexpr int V = VN<T>::N;
    auto kern = k_resid_restrict_z<T, R, HAS_RHS>;
    static PerDevice slots_pd;
    const int slots = per_device(slots_pd, c, [&] {
        prefer_l1(kern);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 128, 0);
        return std::max(1, nb) * c->num_sms;
    });
    const long long items = (long long)((f.sy + R - 1) / R) * (f.sx / V);
    const long long warps = (items + 1 + 30) / 31;   // lanes 1..31 of each warp carry items
    const long long xb = (warps + 3) / 4;
    const int planes = co.nz - 2;
    const int nzc = pick_chunks(xb, planes, slots, R == 2 ? 1 : 4);
    const int Kchunk = (planes + nzc - 1) / nzc;
    const int nzc2 = (planes + Kchunk - 1) / Kchunk;
    dim3 grid((unsigned)xb, (unsigned)nzc2);
    launch_pdl(c, kern, grid, dim3(128), 0, lp_of<T>(c, f), (const T*)u, (const T*)rhs, co.sx, co.sp, co.nz, (T*)rc, Kchunk, nzc2, reverse, done);
}

void launch_resid_restrict_z(mhs_ctx* c, const Level& f, const void* u, const void* rhs, const Level& co, void* rc, int reverse, const int* done)
{
    count_launch(c);
    const bool mid = mid_level(c, f);
#define RR(T)                                                                                  \
    do {                                                                                       \
        if (mid) {                                                                             \
            if (rhs) resid_restrict_t<T, 2, true>(c, f, u, rhs, co, rc, reverse, done);        \
            else resid_restrict_t<T, 2, false>(c, f, u, rhs, co, rc, reverse, done);           \
        } else {                                                                               \
            if (rhs) resid_restrict_t<T, 4, true>(c, f, u, rhs, co, rc, reverse, done);        \
            else resid_restrict_t<T, 4, false>(c, f, u, rhs, co, rc, reverse, done);           \
        }                                                                                      \
    } while (0)
    if (c->es == 8) RR(double);
    else RR(float);
#undef RR
}

void launch_prolong_v(mhs_ctx* c, const Level& f, void* u, const Level& co, const void* ec, int reverse, const int* done)
{
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_prolong_v<double>); prefer_l1(k_prolong_v<float>); return 1; });
    count_launch(c);
    const int V = c->es == 8 ? 2 : 4;
    dim3 grid((unsigned)((f.sp / V + 255) / 256), (unsigned)(f.nz - 2));
    if (c->es == 8)
        launch_pdl(c, k_prolong_v<double>, grid, dim3(256), 0, f.sx, f.sy, f.sp, (double*)u, co.sx, co.sp, (const double*)ec, reverse, f.nz - 2, done);
    else
        launch_pdl(c, k_prolong_v<float>, grid, dim3(256), 0, f.sx, f.sy, f.sp, (float*)u, co.sx, co.sp, (const float*)ec, reverse, f.nz - 2, done);
}

// ------------------------------------------------------------------------------------------------
// Residual + full weighting of a BIG level in separable form (a3 + a4).  Every operator involved is a tensor
// product, and the 27 fine nodes under a coarse interior node are all interior, so
//     R (f - L u) = R f - [ Rz c_k ( (Rx Dxx) (x) Ry + Rx (x) (Ry Dyy) ) + (Rx (x) Ry) (Rz Dzz) + a^2 Rx (x) Ry (x) Rz ] u
// with the 1D composites  R = (1/4, 1/2, 1/4) on offsets (-1, 0, 1)  and  R D2 = (1/4, -1/2, 1/4) / h^2 on offsets
// (-2, 0, 2).  A thread reduces each fine row it touches in x to two numbers, scatters them into the y-partials of
// its RC coarse rows, and scatters those into a sliding window of three coarse planes while it walks up in z: no plane
// of u is kept, the residual is never formed, ~6 flops per fine node instead of ~15.  Same result as residual-then-
// restrict up to rounding order (the sums are regrouped, rounding-order differences).
// Work item: x vector xv (V fine columns -> V/2 coarse columns), coarse rows J0 .. J0+RC-1.
// ------------------------------------------------------------------------------------------------
template <typename T, int RC, bool HAS_RHS>
__global__ void __launch_bounds__(128) k_resid_restrict_sep(LP<T> p, const T* __restrict__ u, const T* __restrict__ rhs, int csx, int csy,
                                                            long long csp, int cnz, T* __restrict__ rc, int Kchunk, int reverse,
                                                            const int* __restrict__ done)
{
    pdl_enter();
    if (done && *done) return;
    constexpr int V = VN<T>::N;
    constexpr int VC = V / 2;
    constexpr int NROW = 2 * RC + 3;
    const int nvx = p.sx / V;
    const int ngroups = (csy - 1 + RC - 1) / RC;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (long long)nvx * ngroups) return;
    const int g = (int)(q / nvx), xv = (int)(q - (long long)g * nvx);
    const int i0 = xv * V, J0 = 1 + g * RC;
    const int zc = reverse ? (int)gridDim.y - 1 - (int)blockIdx.y : (int)blockIdx.y;
    const int Kb = 1 + zc * Kchunk;
    const int Ke = min(Kb + Kchunk, cnz - 1);
    if (Kb >= Ke) return;
    const T hz2 = p.cz, a2 = p.a2;                       // 1/hz^2, alpha^2
    const T* tab = p.tab;                                // cx[k] = c_k/hx^2 | cy[k] = c_k/hy^2
    const long long rowbase = i0 + (long long)p.sx * (2 * J0 - 2);

    T accM[RC][VC], accC[RC][VC], accP[RC][VC];          // coarse planes K-1, K, K+1 of  R L u
    T fC[RC][VC], fP[RC][VC];                            // coarse planes K, K+1 of  R f
#pragma unroll
    for (int s = 0; s < RC; ++s)
#pragma unroll
        for (int m = 0; m < VC; ++m) accM[s][m] = accC[s][m] = accP[s][m] = fC[s][m] = fP[s][m] = T(0);

    // xy-reduced quantities of fine plane k for the thread's coarse nodes:  A = (Rx Ry) u,  Q = c_k (RxDxx Ry + Rx RyDyy) u,  F = (Rx Ry) f
    auto plane = [&](int k, T (&A)[RC][VC], T (&Q)[RC][VC], T (&F)[RC][VC]) {
        T Bx[RC][VC], By[RC][VC];
#pragma unroll
        for (int s = 0; s < RC; ++s)
#pragma unroll
            for (int m = 0; m < VC; ++m) A[s][m] = Bx[s][m] = By[s][m] = F[s][m] = T(0);
        const T* pl = u + rowbase + p.sp * k;
#pragma unroll
        for (int t = 0; t < NROW; ++t) {
            const T* row = pl + (long long)p.sx * t;
            const Vec<T> c = ldv(row);
            const T l0 = row[-2], l1 = row[-1], r0 = row[V];
            T a[VC], b[VC];
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                const T um2 = m == 0 ? l0 : c.v[2 * m - 2], um1 = m == 0 ? l1 : c.v[2 * m - 1];
                const T up1 = c.v[2 * m + 1], up2 = m == VC - 1 ? r0 : c.v[2 * m + 2];
                a[m] = T(0.5) * c.v[2 * m] + T(0.25) * (um1 + up1);
                b[m] = T(0.25) * (um2 + up2) - T(0.5) * c.v[2 * m];
            }
            T af[VC];
            if (HAS_RHS && t >= 1 && t <= NROW - 2) {
                const T* fr = rhs + rowbase + p.sp * k + (long long)p.sx * t;
                const Vec<T> f = ldv(fr);
                const T fl = fr[-1];
#pragma unroll
                for (int m = 0; m < VC; ++m) af[m] = T(0.5) * f.v[2 * m] + T(0.25) * ((m == 0 ? fl : f.v[2 * m - 1]) + f.v[2 * m + 1]);
            }
#pragma unroll
            for (int s = 0; s < RC; ++s) {
                const int d = t - (2 + 2 * s);   // fine row offset from the coarse row's centre
#pragma unroll
                for (int m = 0; m < VC; ++m) {
                    if (d == 0) { A[s][m] += T(0.5) * a[m]; Bx[s][m] += T(0.5) * b[m]; By[s][m] -= T(0.5) * a[m]; }
                    if (d == 1 || d == -1) { A[s][m] += T(0.25) * a[m]; Bx[s][m] += T(0.25) * b[m]; }
                    if (d == 2 || d == -2) By[s][m] += T(0.25) * a[m];
                    if (HAS_RHS) {
                        if (d == 0) F[s][m] += T(0.5) * af[m];
                        if (d == 1 || d == -1) F[s][m] += T(0.25) * af[m];
                    }
                }
            }
        }
        const T cx = tab[k], cy = tab[p.nz + k];
#pragma unroll
        for (int s = 0; s < RC; ++s)
#pragma unroll
            for (int m = 0; m < VC; ++m) Q[s][m] = cx * Bx[s][m] + cy * By[s][m];
    };

    for (int K = Kb - 1; K <= Ke; ++K) {
        T A[RC][VC], Q[RC][VC], F[RC][VC];
        // even fine plane 2K: weight 1/2 for K; its (Rz Dzz) part also feeds K-1 and K+1
        plane(2 * K, A, Q, F);
        const bool zin = 2 * K >= 1 && 2 * K <= p.nz - 2;   // L u (and f) live on interior planes only
#pragma unroll
        for (int s = 0; s < RC; ++s)
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                const T az = T(0.25) * hz2 * A[s][m];
                accM[s][m] += az;
                accP[s][m] += az;
                accC[s][m] += (zin ? T(0.5) * Q[s][m] + T(0.5) * a2 * A[s][m] : T(0)) - T(0.5) * hz2 * A[s][m];
                if (HAS_RHS && zin) fC[s][m] += T(0.5) * F[s][m];
            }
        // coarse plane K-1 is complete
        if (K - 1 >= Kb) {
#pragma unroll
            for (int s = 0; s < RC; ++s)
#pragma unroll
                for (int m = 0; m < VC; ++m) {
                    const int I = (i0 >> 1) + m, J = J0 + s;
                    if (I > 0 && J < csy) rc[I + (long long)csx * J + csp * (K - 1)] = -accM[s][m];
                }
        }
        if (K == Ke) break;
        // odd fine plane 2K+1: weight 1/4 for K and for K+1
        plane(2 * K + 1, A, Q, F);
#pragma unroll
        for (int s = 0; s < RC; ++s)
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                const T v = T(0.25) * Q[s][m] + T(0.25) * a2 * A[s][m];
                accC[s][m] += v;
                accP[s][m] += v;
                if (HAS_RHS) { fC[s][m] += T(0.25) * F[s][m]; fP[s][m] += T(0.25) * F[s][m]; }
            }
        // slide the window: K -> K+1.  (R f)[K] is complete here too; fold it into the plane that is stored next.
#pragma unroll
        for (int s = 0; s < RC; ++s)
#pragma unroll
            for (int m = 0; m < VC; ++m) {
                accM[s][m] = HAS_RHS ? accC[s][m] - fC[s][m] : accC[s][m];
                accC[s][m] = accP[s][m];
                accP[s][m] = T(0);
                fC[s][m] = fP[s][m];
                fP[s][m] = T(0);
            }
    }
}

template <typename T, bool HAS_RHS, int RC>
static void resid_restrict_sep_t(mhs_ctx* c, const Level& f, const void* u, const void* rhs, const Level& co, void* rc, int reverse, const int* done)
{
    constexpr int V = VN<T>::N;
    auto kern = k_resid_restrict_sep<T, RC, HAS_RHS>;
    static PerDevice slots_pd;
    const int slots = per_device(slots_pd, c, [&] {
        prefer_l1(kern);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 128, 0);
        return std::max(1, nb) * c->num_sms;
    });
    const long long items = (long long)(f.sx / V) * ((co.sy - 1 + RC - 1) / RC);
    const long long xb = (items + 127) / 128;
    const int planes = co.nz - 2;
    // z-chunks: one wave of resident blocks (the kernel is bound by parallelism before bytes: measured at 257^3, 32 chunks
    // of 4 coarse planes -- 11 fine planes read for 8 -- beat 16 chunks of 8 by 57 -> 41 us); no shorter than 4 coarse planes
    const int minlen = 4;
    int nzc = (int)std::max<long long>(1, std::min<long long>(planes / minlen > 0 ? planes / minlen : 1, slots / xb));
    const int Kchunk = (planes + nzc - 1) / nzc;
    nzc = (planes + Kchunk - 1) / Kchunk;
    dim3 grid((unsigned)xb, (unsigned)nzc);
    launch_pdl(c, kern, grid, dim3(128), 0, lp_of<T>(c, f), (const T*)u, (const T*)rhs, co.sx, co.sy, co.sp, co.nz, (T*)rc, Kchunk, reverse, done);
}

void launch_resid_restrict_sep(mhs_ctx* c, const Level& f, const void* u, const void* rhs, const Level& co, void* rc, int reverse, const int* done)
{
    count_launch(c);
    // (only big levels come here -- mhs_api.cu restrict_fast; two coarse rows per thread, RC = 2, measured no faster)
#define RS(T)                                                                                    \
    do {                                                                                         \
        if (rhs) resid_restrict_sep_t<T, true, 4>(c, f, u, rhs, co, rc, reverse, done);          \
        else resid_restrict_sep_t<T, false, 4>(c, f, u, rhs, co, rc, reverse, done);             \
    } while (0)
    if (c->es == 8) RS(double);
    else RS(float);
#undef RS
}

}  // namespace mhs
