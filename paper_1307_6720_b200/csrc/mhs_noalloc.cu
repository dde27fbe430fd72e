// mhs_resnorm_static: the residual norm of eq 8 (stop rule C10) for callers that may not allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It is a variant of the
// residual-norm kernel (k_resnorm_partial_ref + k_norm_final, which keep their partial sums in a buffer that mhs_create
// allocates) with the partial sums in a FILE-SCOPE device array instead: no context, no cudaMalloc / cudaFree, no
// allocating library routine.  Every GPU that loads the library holds the array (512 KB) until the process exits.
//
// The array is shared by every call: calls that overlap on the GPU (two streams, two host threads) race on it.  It keeps
// the last call's contents; nothing in it has to start at zero, because every element a call reads (partials 0 .. n-1)
// is written by that same call first -- the reduction kernel never looks beyond n.
#include <atomic>
#include <cstdio>
#include <string>

#include "mhs_device.cuh"

namespace mhs {

static __device__ __align__(256) double g_static_scratch[MHS_STATIC_SCRATCH_DOUBLES];

constexpr int NA_ROWS = 8;   // rows of one plane per block = per partial sum

// partial[b] = sum over the block's interior nodes of (L P)^2; dense layout, idx = i + nx (j + ny k)
template <typename T>
__global__ void __launch_bounds__(256) k_resnorm_static_partial(const T* __restrict__ P, const double* __restrict__ c, int nx, int ny, int nz,
                                                                double hx2, double hy2, double i_hz2, double a2d, double* __restrict__ partial)
{
    const int k = 1 + (int)blockIdx.y;
    const int j = 1 + (int)blockIdx.x * NA_ROWS + (int)threadIdx.y;
    double acc = 0.0;
    if (j < ny - 1) {
        // the coefficients as the solver's tables hold them: formed in fp64, rounded to T once
        const T cx = (T)(c[k] / hx2), cy = (T)(c[k] / hy2), cz = (T)i_hz2, a2 = (T)a2d;
        const long long sp = (long long)nx * ny;
        const T* row = P + (long long)nx * j + sp * k;
        for (int i = 1 + (int)threadIdx.x; i < nx - 1; i += 32) {
            const T uc = row[i];
            T lu = cx * lap1<T>(row[i + 1], row[i - 1], uc) + cy * lap1<T>(row[i + nx], row[i - nx], uc);
            lu += cz * lap1<T>(row[i + sp], row[i - sp], uc) + a2 * uc;
            const double r = (double)(T(0) - lu);   // rhs = 0: eq 8 is homogeneous
            acc += r * r;
        }
    }
    acc = block_sum<256>(acc);
    if (threadIdx.x == 0 && threadIdx.y == 0) partial[blockIdx.y * gridDim.x + blockIdx.x] = acc;
}

// out = sqrt(sum of partial[0 .. n-1]), summed in a fixed order (the result does not depend on scheduling)
__global__ void __launch_bounds__(1024) k_resnorm_static_final(const double* __restrict__ partial, int n, double* __restrict__ out)
{
    double acc = 0.0;
    for (int q = threadIdx.x; q < n; q += 1024) acc += partial[q];
    acc = block_sum<1024>(acc);
    if (threadIdx.x == 0) *out = sqrt(acc);
}

static thread_local std::string t_static_err;

static mhs_status static_fail(mhs_status st, const std::string& msg)
{
    t_static_err = msg;
    return st;
}

// The device address of the scratch array, once per device.  In host code `g_static_scratch` is a host-side stand-in
// for the symbol, not a device address: the kernels must be given what cudaGetSymbolAddress returns for the device
// that is current.
static mhs_status static_scratch_address(double** out)
{
    static std::atomic<double*> addr[MAX_DEVICES];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(MHS_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return static_fail(MHS_ERR_CUDA, "device ordinal out of range");
    double* p = addr[dev].load(std::memory_order_acquire);
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess || !p) return static_fail(MHS_ERR_CUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
        addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return MHS_OK;
}

}  // namespace mhs

using namespace mhs;

extern "C" {

const char* mhs_static_last_error(void) { return t_static_err.c_str(); }

mhs_status mhs_resnorm_static(const void* P_device, int dtype, int nx, int ny, int nz, double hx, double hy, double hz, double alpha,
                              const double* c_device, double* out_device, void* stream)
{
    if (!P_device || !c_device || !out_device) return static_fail(MHS_ERR_INVALID_ARG, "mhs_resnorm_static: null pointer");
    if (dtype != MHS_F32 && dtype != MHS_F64) return static_fail(MHS_ERR_INVALID_ARG, "mhs_resnorm_static: dtype must be MHS_F32 or MHS_F64");
    if (nx < 3 || ny < 3 || nz < 3) return static_fail(MHS_ERR_INVALID_ARG, "mhs_resnorm_static: every extent must be >= 3");
    if (!(hx > 0.0) || !(hy > 0.0) || !(hz > 0.0)) return static_fail(MHS_ERR_INVALID_ARG, "mhs_resnorm_static: mesh widths must be positive");
    const long long gx = (ny - 2 + NA_ROWS - 1) / NA_ROWS, gy = nz - 2;
    const long long need = gx * gy;
    if (need > MHS_STATIC_SCRATCH_DOUBLES || gy > 65535) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "mhs_resnorm_static: a %d x %d x %d grid needs %lld partial sums (ceil((ny-2)/%d) * (nz-2)); the static scratch array holds "
                 "MHS_STATIC_SCRATCH_DOUBLES = %d",
                 nx, ny, nz, need, NA_ROWS, MHS_STATIC_SCRATCH_DOUBLES);
        return static_fail(MHS_ERR_INVALID_ARG, msg);
    }
    double* scratch = nullptr;
    { mhs_status st = static_scratch_address(&scratch); if (st) return st; }
    cudaStream_t s = (cudaStream_t)stream;
    const dim3 grid((unsigned)gx, (unsigned)gy), block(32, NA_ROWS);
    const double hx2 = hx * hx, hy2 = hy * hy, ihz2 = 1.0 / (hz * hz), a2 = alpha * alpha;
    if (dtype == MHS_F64)
        k_resnorm_static_partial<double><<<grid, block, 0, s>>>((const double*)P_device, c_device, nx, ny, nz, hx2, hy2, ihz2, a2, scratch);
    else
        k_resnorm_static_partial<float><<<grid, block, 0, s>>>((const float*)P_device, c_device, nx, ny, nz, hx2, hy2, ihz2, a2, scratch);
    k_resnorm_static_final<<<1, 1024, 0, s>>>(scratch, (int)need, out_device);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(MHS_ERR_CUDA, std::string("mhs_resnorm_static launch: ") + cudaGetErrorString(e));
    return MHS_OK;
}

}  // extern "C"
