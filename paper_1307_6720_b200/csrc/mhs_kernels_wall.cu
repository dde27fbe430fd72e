// Non-zero Dirichlet data for P on the side and top faces ("In principle other elliptic
// equations can be defined on the other boundaries" -- whatever they give is Dirichlet data for eq 8 on those faces).
//
// The solver's arrays store every side/top wall value once and as zero (the aliased layout, mhs_internal.h), and every kernel
// relies on that.  Wall data therefore enters by LIFTING: with W = the data on the side/top wall nodes and zero everywhere
// else, P = P_h + W where P_h has zero walls and solves  L P_h = -L W  in the interior -- a right-hand side that is non-zero
// only at the interior nodes next to a wall.  The finest level gets a right-hand side array for it and runs the kernels the
// coarser levels run (they all take one); results leave the library as P_h + W.
//   k_wall_take : caller's dense array -> W (wall nodes kept, everything else zero; faces declared MHS_BC_DIRICHLET_ZERO zero)
//   k_wall_rhs  : rhs0 = -L W at the interior nodes (aliased layout)
//   k_wall_add  : dense P += W
#include "mhs_device.cuh"

namespace mhs {

template <typename T>
__global__ void __launch_bounds__(256) k_wall_take(int nx, int ny, int nz, int sides, int top, const T* __restrict__ G, T* __restrict__ W)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= nx || j >= ny) return;
    const bool side = i == 0 || j == 0 || i == nx - 1 || j == ny - 1;
    const bool tp = !side && k == nz - 1;
    const long long d = i + (long long)nx * (j + (long long)ny * k);
    W[d] = (side && sides) || (tp && top) ? G[d] : T(0);
}

// tab: cx[nz] | cy[nz] | ... of the finest level (cx = c_k / hx^2); cz = 1 / hz^2
template <typename T>
__global__ void __launch_bounds__(256) k_wall_rhs(int nx, int ny, int nz, int sx, long long sp, const T* __restrict__ tab, T cz,
                                                  const T* __restrict__ W, T* __restrict__ rhs)
{
    const int i = 1 + blockIdx.x * blockDim.x + threadIdx.x;
    const int j = 1 + blockIdx.y * blockDim.y + threadIdx.y;
    const int k = 1 + blockIdx.z;
    if (i >= nx - 1 || j >= ny - 1) return;
    const long long py = nx, pz = (long long)nx * ny;
    const T* w = W + i + py * j + pz * k;
    // (W is zero at every node that is not a side or top wall node, the bottom plane's interior included)
    const T lw = tab[k] * (w[1] + w[-1]) + tab[nz + k] * (w[py] + w[-py]) + cz * (w[pz] + w[-pz]);
    rhs[i + (long long)sx * j + sp * k] = -lw;
}

template <typename T>
__global__ void __launch_bounds__(256) k_wall_add(long long n, const T* __restrict__ W, T* __restrict__ P)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) P[q] += W[q];
}

void launch_wall_take(mhs_ctx* c, const Level& lv, int sides, int top, const void* G, void* W)
{
    const dim3 b(32, 8), g((lv.nx + 31) / 32, (lv.ny + 7) / 8, lv.nz);
    count_launch(c);
    if (c->es == 8) k_wall_take<double><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, sides, top, (const double*)G, (double*)W);
    else k_wall_take<float><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, sides, top, (const float*)G, (float*)W);
}

void launch_wall_rhs(mhs_ctx* c, const Level& lv, const void* W, void* rhs)
{
    const dim3 b(32, 8), g((lv.nx - 2 + 31) / 32, (lv.ny - 2 + 7) / 8, lv.nz - 2);
    count_launch(c);
    const double cz = 1.0 / (lv.hz * lv.hz);
    if (c->es == 8)
        k_wall_rhs<double><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, lv.sx, lv.sp, (const double*)lv.tab, cz, (const double*)W, (double*)rhs);
    else
        k_wall_rhs<float><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, lv.sx, lv.sp, (const float*)lv.tab, (float)cz, (const float*)W, (float*)rhs);
}

void launch_wall_add(mhs_ctx* c, const Level& lv, const void* W, void* P)
{
    const long long n = lv.npts();
    count_launch(c);
    if (c->es == 8) k_wall_add<double><<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, (const double*)W, (double*)P);
    else k_wall_add<float><<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, (const float*)W, (float*)P);
}

}  // namespace mhs
