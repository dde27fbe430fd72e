// Device helpers shared by the kernels of libmhs_b200.
#pragma once
#include "mhs_internal.h"

namespace mhs {

// a + b - 2c, the numerator of a compact second difference.  fp64: one add + one FMA.  fp32: the
// difference form (a-c)+(b-c), whose rounding error scales with the differences instead of with
// |u| -- it lowers the fp32 residual floor.
template <typename T>
__device__ __forceinline__ T lap1(T a, T b, T c);
template <>
__device__ __forceinline__ double lap1<double>(double a, double b, double c) { return fma(-2.0, c, a + b); }
template <>
__device__ __forceinline__ float lap1<float>(float a, float b, float c) { return (a - c) + (b - c); }

// (L u) at the interior node with linear index c on plane k:
//   c_k/hx^2 dxx + c_k/hy^2 dyy + 1/hz^2 dzz + alpha^2 u      (eq 8; 2D: eq 11, :94)
template <typename T, bool D3>
__device__ __forceinline__ T apply_L(const LP<T>& p, const T* __restrict__ u, long long c, int k)
{
    const T uc = u[c];
    T lu = p.tab[k] * lap1<T>(u[c + 1], u[c - 1], uc) + p.tab[p.nz + k] * lap1<T>(u[c + p.sx], u[c - p.sx], uc);
    if (D3) lu += p.cz * lap1<T>(u[c + p.sp], u[c - p.sp], uc) + p.a2 * uc;
    return lu;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over a block of NT threads (any block shape); the result is valid in thread 0.
template <int NT>
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double s_part[NT / 32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    v = warp_sum(v);
    if ((tid & 31) == 0) s_part[tid >> 5] = v;
    __syncthreads();
    if (tid < 32) {
        double w = tid < NT / 32 ? s_part[tid] : 0.0;
        w = warp_sum(w);
        v = w;
    }
    return v;
}

}  // namespace mhs
