// Field-line integration of libmhs_b200 (the field lines of the paper's Figs 1, 4, 5,
// PAPER.md:142-144, :158-186):   dx/ds = dir * B(x) / |B(x)|,  B between the nodes by trilinear interpolation of the
// dense nodal B that mhs_fields wrote, classical RK4 with a fixed arc-length step, polylines into a device buffer.
//
// One thread per line.  A step is four samples x three components x eight corners = 96 gathers, all independent within
// a stage, from the 3N-word B array (at 257^3 fp64: 407 MB, larger than the L2; neighbouring seeds share cells and
// lines stay inside a few planes for many steps, so most gathers hit L1/L2).  The kernel is bound by the latency of a
// chain of dependent gathers (4 stages per step, steps strictly sequential), not by bytes: parallelism = number of seeds.
// fp64 evaluates every product-sum as an fma in a fixed order (mhs.h documents it) so that a CPU implementation that
// does the same gets the same points bit for bit -- the exit tests decide an integer.
#include "mhs_device.cuh"

namespace mhs {

template <typename T>
struct LineP {
    int nx, ny, nz;
    long long sy, sz;       // dense strides: nx, nx*ny
    T Lx, Ly, Lz, ihx, ihy, ihz;
    T h, h2, h6, dir, bmin;
    int max_points, nseeds;
};

template <typename T> __device__ __forceinline__ T fma_t(T a, T b, T c);
template <> __device__ __forceinline__ double fma_t<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fma_t<float>(float a, float b, float c) { return fmaf(a, b, c); }

// a product that must stay a product (never fused into a following add)
__device__ __forceinline__ double mul_t(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_t(float a, float b) { return __fmul_rn(a, b); }

template <typename T>
__device__ __forceinline__ bool inside(const LineP<T>& p, T x, T y, T z)
{
    return x >= T(0) && x <= p.Lx && y >= T(0) && y <= p.Ly && z >= T(0) && z <= p.Lz;
}

// unit tangent dir * B / |B| at (x, y, z); false: outside the box or |B| <= bmin
template <typename T>
__device__ __forceinline__ bool tangent(const LineP<T>& p, const T* __restrict__ Bx, const T* __restrict__ By, const T* __restrict__ Bz, T x,
                                        T y, T z, T (&t)[3])
{
    if (!inside(p, x, y, z)) return false;
    const T fx = mul_t(x, p.ihx), fy = mul_t(y, p.ihy), fz = mul_t(z, p.ihz);
    int i = (int)floor(fx), j = (int)floor(fy), k = (int)floor(fz);
    i = max(0, min(i, p.nx - 2)); j = max(0, min(j, p.ny - 2)); k = max(0, min(k, p.nz - 2));
    const T tx = fx - (T)i, ty = fy - (T)j, tz = fz - (T)k;
    const long long q = i + p.sy * j + p.sz * k;
    T b[3];
    const T* comp[3] = {Bx, By, Bz};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T* a = comp[c] + q;
        const T a000 = __ldg(a), a100 = __ldg(a + 1), a010 = __ldg(a + p.sy), a110 = __ldg(a + p.sy + 1);
        const T a001 = __ldg(a + p.sz), a101 = __ldg(a + p.sz + 1), a011 = __ldg(a + p.sz + p.sy), a111 = __ldg(a + p.sz + p.sy + 1);
        const T b00 = fma_t<T>(tx, a100 - a000, a000), b10 = fma_t<T>(tx, a110 - a010, a010);
        const T b01 = fma_t<T>(tx, a101 - a001, a001), b11 = fma_t<T>(tx, a111 - a011, a011);
        const T c0 = fma_t<T>(ty, b10 - b00, b00), c1 = fma_t<T>(ty, b11 - b01, b01);
        b[c] = fma_t<T>(tz, c1 - c0, c0);
    }
    const T m = sqrt(fma_t<T>(b[2], b[2], fma_t<T>(b[1], b[1], mul_t(b[0], b[0]))));
    if (!(m > p.bmin)) return false;
    const T s = p.dir / m;
    t[0] = mul_t(b[0], s); t[1] = mul_t(b[1], s); t[2] = mul_t(b[2], s);
    return true;
}

template <typename T>
__global__ void __launch_bounds__(128) k_fieldlines(const LineP<T> p, const T* __restrict__ Bx, const T* __restrict__ By,
                                                    const T* __restrict__ Bz, const T* __restrict__ seeds, T* __restrict__ lines,
                                                    int* __restrict__ npoints)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= p.nseeds) return;
    T x = seeds[3 * s], y = seeds[3 * s + 1], z = seeds[3 * s + 2];
    T* out = lines + (long long)s * p.max_points * 3;
    int n = 0;
    if (p.max_points > 0 && inside(p, x, y, z)) {
        out[0] = x; out[1] = y; out[2] = z;
        n = 1;
        while (n < p.max_points) {
            T k1[3], k2[3], k3[3], k4[3];
            if (!tangent(p, Bx, By, Bz, x, y, z, k1)) break;
            if (!tangent(p, Bx, By, Bz, fma_t<T>(p.h2, k1[0], x), fma_t<T>(p.h2, k1[1], y), fma_t<T>(p.h2, k1[2], z), k2)) break;
            if (!tangent(p, Bx, By, Bz, fma_t<T>(p.h2, k2[0], x), fma_t<T>(p.h2, k2[1], y), fma_t<T>(p.h2, k2[2], z), k3)) break;
            if (!tangent(p, Bx, By, Bz, fma_t<T>(p.h, k3[0], x), fma_t<T>(p.h, k3[1], y), fma_t<T>(p.h, k3[2], z), k4)) break;
            const T xn = fma_t<T>(p.h6, (k1[0] + k4[0]) + T(2) * (k2[0] + k3[0]), x);
            const T yn = fma_t<T>(p.h6, (k1[1] + k4[1]) + T(2) * (k2[1] + k3[1]), y);
            const T zn = fma_t<T>(p.h6, (k1[2] + k4[2]) + T(2) * (k2[2] + k3[2]), z);
            if (!inside(p, xn, yn, zn)) break;
            x = xn; y = yn; z = zn;
            out[3 * n] = x; out[3 * n + 1] = y; out[3 * n + 2] = z;
            ++n;
        }
    }
    npoints[s] = n;
}

template <typename T>
static void fieldlines_t(mhs_ctx* c, const Level& lv, const void* B, int nseeds, const void* seeds, double step, int max_points,
                         int direction, double bmin, void* lines, int* npoints)
{
    LineP<T> p;
    p.nx = lv.nx; p.ny = lv.ny; p.nz = lv.nz;
    p.sy = lv.nx; p.sz = (long long)lv.nx * lv.ny;
    p.Lx = (T)c->grid.Lx; p.Ly = (T)c->grid.Ly; p.Lz = (T)c->grid.Lz;
    // (nx-1)/Lx etc. in double, then rounded: the same numbers a double-precision caller computes
    p.ihx = (T)((lv.nx - 1) / c->grid.Lx); p.ihy = (T)((lv.ny - 1) / c->grid.Ly); p.ihz = (T)((lv.nz - 1) / c->grid.Lz);
    p.h = (T)step; p.h2 = (T)(0.5 * step); p.h6 = (T)(step / 6.0);
    p.dir = direction < 0 ? T(-1) : T(1);
    p.bmin = (T)bmin;
    p.max_points = max_points; p.nseeds = nseeds;
    const long long N = lv.npts();
    const T* Bp = (const T*)B;
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_fieldlines<T>); return 1; });
    k_fieldlines<T><<<(nseeds + 127) / 128, 128, 0, c->stream>>>(p, Bp, Bp + N, Bp + 2 * N, (const T*)seeds, (T*)lines, npoints);
}

void launch_fieldlines(mhs_ctx* c, const Level& lv, const void* B, int nseeds, const void* seeds, double step, int max_points, int direction,
                       double bmin, void* lines, int* npoints)
{
    count_launch(c);
    if (c->es == 8) fieldlines_t<double>(c, lv, B, nseeds, seeds, step, max_points, direction, bmin, lines, npoints);
    else fieldlines_t<float>(c, lv, B, nseeds, seeds, step, max_points, direction, bmin, lines, npoints);
}

}  // namespace mhs
