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

// Programmatic dependent launch (PDL): the kernels of a cycle are a chain of small dependent launches, and on the levels
// that live in the L2 launch latency is most of their time.  Every kernel starts with pdl_enter(): it lets the NEXT kernel
// of the stream be scheduled as soon as all blocks of this one are running (its blocks then sit in their own pdl_enter),
// and it waits until the PREVIOUS kernel has completed and its writes are visible.  Nothing that depends on earlier
// kernels (not even the `done` flag) may be touched before it.  Without the launch attribute both are no-ops.
__device__ __forceinline__ void pdl_enter()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
// The two halves, for a kernel with work that does not depend on its predecessors (the cluster kernel zeroes its shared
// memory and copies constant tables in between).
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

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

// Stop rule (C10, C20), evaluated by ONE thread with the freshly reduced residual norm r.
//   mode 1: r is the residual of the iterate reached after ctl->units completed cycles.
//           units == 0: this is r0 (kept if the caller already knew it);  otherwise record cycle `units`
//           and apply the stop rule.  If the solve goes on, units is advanced: the rest of the cycle may run.
//   mode 2: r_last only (operator-level queries).
__device__ __forceinline__ void stop_rule(Ctl* ctl, double r, int mode)
{
    if (mode == 2) {
        ctl->r_last = r;
        return;
    }
    const int k = ctl->units;
    const bool bad = !(r == r) || isinf(r);
    if (bad) ctl->nan_seen = 1;
    if (k == 0) {
        if (!(ctl->r0 > 0.0)) ctl->r0 = r;
        ctl->r_last = r;
        if (bad) ctl->done = 1;
    } else {
        const double prev = ctl->r_last;
        if (k - 1 < MHS_HISTORY_LEN) ctl->hist[k - 1] = r;
        ctl->cycles = k;
        ctl->r_last = r;
        bool stag = false;
        if (ctl->stag_on) {  // C20: the fp32 residual floor shows as r_k > 0.9 r_{k-1} twice in a row
            ctl->stag_count = (r > 0.9 * prev) ? ctl->stag_count + 1 : 0;
            stag = ctl->stag_count >= 2;
            if (stag) ctl->stagnated = 1;
        }
        if (bad || stag || r <= ctl->tol * ctl->r0 || k >= ctl->max_cycles) ctl->done = 1;
    }
    if (!ctl->done) ctl->units = k + 1;
}

}  // namespace mhs
