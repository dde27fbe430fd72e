// Residual + full weighting of the finest (HBM-bound) level as a bulk-copy fed streaming kernel (a3 + a4).
//
// Same arithmetic as k_resid_restrict_sep (mhs_kernels_fast.cu): the separable form
//     R (0 - L u) = -[ Rz c_k ( (Rx Dxx) (x) Ry + Rx (x) (Ry Dyy) ) + (Rx (x) Ry) (Rz Dzz) + a^2 Rx (x) Ry (x) Rz ] u ,
// R = (1/4, 1/2, 1/4) on offsets (-1, 0, 1), R D2 = (1/4, -1/2, 1/4)/h^2 on offsets (-2, 0, 2): every fine plane is reduced
// in x and y to two coarse-resolution numbers per coarse node, and those are scattered over a sliding window of three coarse
// planes while the kernel walks through z.  What differs is how the data arrive.  That kernel loads through the L1 and was
// bound by DRAM latency (44 us at 257^3 for 153 MB: 3.5 TB/s, `long_scoreboard`); here a CTA owns a strip of RC*G coarse
// rows x all columns, the 2 RC G + 3 fine rows under it are ONE contiguous chunk of each plane in the aliased layout, and
// they are brought in by the bulk-copy engine (cp.async.bulk, completion on mbarriers) into a ring of planes several planes
// ahead of the arithmetic -- the data path of k_zsweep -- so that the pass runs at the speed of the memory.
// The walk goes DOWN in z on request: the smoothing pass that wrote u finished every z-segment at its top, so the planes
// written last -- the ones still in the L2 -- are read first.
#include <algorithm>
#include <cstdint>

#include "mhs_device.cuh"

namespace mhs {

namespace {

__device__ __forceinline__ uint32_t rr_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void rr_bar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(rr_smem(bar)), "r"(count));
}
__device__ __forceinline__ void rr_expect(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(rr_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void rr_bulk(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(rr_smem(dst)), "l"(src),
                 "r"(bytes), "r"(rr_smem(bar))
                 : "memory");
}
__device__ __forceinline__ void rr_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "RR_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra RR_DONE;\n"
        "bra RR_WAIT;\n"
        "RR_DONE:\n"
        "}\n" ::"r"(rr_smem(bar)),
        "r"(parity)
        : "memory");
}

template <typename T>
struct __align__(2 * sizeof(T)) Pair {
    T a, b;
};

#ifndef MHS_RR_RC
#define MHS_RR_RC 4
#endif
#ifndef MHS_RR_NT
#define MHS_RR_NT 256
#endif
constexpr int RR_RC = MHS_RR_RC;       // coarse rows per thread
#ifndef MHS_RR_RINGCAP
#define MHS_RR_RINGCAP 6
#endif
#ifndef MHS_RR_CPS
#define MHS_RR_CPS 1
#endif
constexpr int RR_MAXRING = MHS_RR_RINGCAP;

template <typename T>
struct RRP {
    int sx, sy, nz;            // fine level: row pitch, rows per plane, planes
    long long sp;
    const T* tab;              // cx[k] | cy[k] | ...
    T hz2, a2;                 // 1/hz^2, alpha^2
    int csx, csy, cnz;         // coarse level
    long long csp;
    int G;                     // thread groups along y: a CTA owns RC*G coarse rows
    int nring;                 // planes of the ring
    int ntiles, nzc;           // strips along y, z-chunks
    int down;                  // walk down in z
    // The cycle's stop rule folded in (instead of a k_norm_final launch between the norm-carrying smoothing pass and this
    // kernel): CTA 0 reduces the norm_n partial sums of the squared residual and applies the rule before its own work.
    const double* norm_partial;
    long long norm_n;          // 0: nothing folded in
    Ctl* ctl;
};

// One CTA: strip `tile` (coarse rows J0 .. J0+RC*G-1), coarse planes [Kb, Ke).
template <typename T>
__global__ void __launch_bounds__(512, 1) k_resid_restrict_ring(const __grid_constant__ RRP<T> p, const T* __restrict__ u, T* __restrict__ rc,
                                                                  const int* __restrict__ done)
{
    constexpr int RC = RR_RC;
    constexpr int NROW = 2 * RC + 3;                       // fine rows under a thread's RC coarse rows
    pdl_enter();
    if (p.norm_n > 0 && blockIdx.x == 0 && !p.ctl->done) {
        // k_norm_final's reduction, sum for sum (1024 virtual threads q, q + 1024, ...; warp sums; their sum in warp 0), so the
        // norms are the same bits whichever kernel forms them.  Every thread has read `done` before thread 0 may raise it
        // (the barrier below).  The other CTAs do not wait for the decision: in the one cycle that finds the tolerance met
        // they restrict a residual nobody uses; every later kernel of that cycle sees the flag.
        __shared__ double s_vw[32];
        for (int t = (int)threadIdx.x; t < 1024; t += (int)blockDim.x) {
            double v = 0.0;
            for (long long q = t; q < p.norm_n; q += 1024) v += p.norm_partial[q];
            v = warp_sum(v);
            if ((t & 31) == 0) s_vw[t >> 5] = v;
        }
        __syncthreads();
        if (threadIdx.x < 32) {
            const double w = warp_sum(s_vw[threadIdx.x]);
            if (threadIdx.x == 0) stop_rule(p.ctl, sqrt(w), 1);
        }
        __syncthreads();
    }
    if (done && *done) return;
    extern __shared__ __align__(128) unsigned char rsm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(rsm);
    T* ring = reinterpret_cast<T*>(rsm + 128);
    const int ncx = p.sx >> 1;                             // coarse columns (threads along x)
    const int I = (int)threadIdx.x % ncx, g = (int)threadIdx.x / ncx;
    const int tile = (int)blockIdx.x % p.ntiles, zc = (int)blockIdx.x / p.ntiles;
    const int J0t = 1 + tile * RC * p.G;                   // first coarse row of the strip
    const int J0 = J0t + g * RC;                           // ... of this thread
    const int planes = p.cnz - 2;
    const int Kb = 1 + (int)((long long)planes * zc / p.nzc), Ke = 1 + (int)((long long)planes * (zc + 1) / p.nzc);
    if (Kb >= Ke) return;
    const int rows_t = 2 * RC * p.G + 3;                   // fine rows of the strip
    const uint32_t slot_elems = (uint32_t)rows_t * p.sx;
    const uint32_t slot_bytes = slot_elems * (uint32_t)sizeof(T);
    // fine planes kf .. kl of the chunk, in walk order
    const int k_lo = 2 * Kb - 2, k_hi = 2 * Ke;
    const int nplanes = k_hi - k_lo + 1;
    const int d = p.down ? -1 : 1;
    const int k_first = p.down ? k_hi : k_lo;
    const T* src0 = u + (long long)p.sx * (2 * J0t - 2);   // (row 2 J0t - 2, column 0) of plane 0

    if (threadIdx.x == 0) {
        for (int q = 0; q < p.nring; ++q) rr_bar_init(bars + q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](int n) {      // plane number n of the walk -> slot n % nring
        const int slot = n % p.nring;
        rr_expect(bars + slot, slot_bytes);
        rr_bulk(ring + (size_t)slot * slot_elems, src0 + p.sp * (k_first + d * n), slot_bytes, bars + slot);
    };
    if (threadIdx.x == 0)
        for (int n = 0; n < min(p.nring, nplanes); ++n) issue(n);

    T accB[RC], accC[RC], accA[RC];                       // coarse planes behind / at / ahead of the walk
#pragma unroll
    for (int s = 0; s < RC; ++s) accB[s] = accC[s] = accA[s] = T(0);
    const T* tab = p.tab;
    const T hz2 = p.hz2, a2 = p.a2;
    // this thread's window inside a slot: fine rows 2 RC g .. 2 RC g + NROW - 1, fine columns 2I-2 .. 2I+2
    const uint32_t own = (uint32_t)(2 * RC * g) * p.sx + 2 * I;

    // xy-reduced quantities of one fine plane for the thread's coarse nodes:  A = (Rx Ry) u,  Q = c_k (RxDxx Ry + Rx RyDyy) u
    auto plane = [&](const T* sl, int k, T (&A)[RC], T (&Q)[RC]) {
        T Bx[RC], By[RC];
#pragma unroll
        for (int s = 0; s < RC; ++s) A[s] = Bx[s] = By[s] = T(0);
        const T* w = sl + own;
#pragma unroll
        for (int t = 0; t < NROW; ++t) {
            const T* row = w + (size_t)t * p.sx;
            const Pair<T> l = *reinterpret_cast<const Pair<T>*>(row - 2);
            const Pair<T> c = *reinterpret_cast<const Pair<T>*>(row);
            const T r0 = row[2];
            const T a = T(0.5) * c.a + T(0.25) * (l.b + c.b);
            const T b = T(0.25) * (l.a + r0) - T(0.5) * c.a;
#pragma unroll
            for (int s = 0; s < RC; ++s) {
                const int dd = t - (2 + 2 * s);   // fine row offset from the coarse row's centre
                if (dd == 0) { A[s] += T(0.5) * a; Bx[s] += T(0.5) * b; By[s] -= T(0.5) * a; }
                if (dd == 1 || dd == -1) { A[s] += T(0.25) * a; Bx[s] += T(0.25) * b; }
                if (dd == 2 || dd == -2) By[s] += T(0.25) * a;
            }
        }
        const T cx = tab[k], cy = tab[p.nz + k];
#pragma unroll
        for (int s = 0; s < RC; ++s) Q[s] = cx * Bx[s] + cy * By[s];
    };

    int n = 0;                                            // planes consumed so far
    auto next_plane = [&](int k, T (&A)[RC], T (&Q)[RC]) {
        const int slot = n % p.nring;
        rr_wait(bars + slot, (uint32_t)((n / p.nring) & 1));
        plane(ring + (size_t)slot * slot_elems, k, A, Q);
        __syncthreads();                                  // everybody is done with the slot
        if (threadIdx.x == 0 && n + p.nring < nplanes) issue(n + p.nring);
        ++n;
    };

    const int K_first = p.down ? Ke : Kb - 1, K_last = p.down ? Kb - 1 : Ke;
    for (int K = K_first;; K += d) {
        T A[RC], Q[RC];
        // even fine plane 2K: weight 1/2 for K; its (Rz Dzz) part also feeds K-1 and K+1
        next_plane(2 * K, A, Q);
        const bool zin = 2 * K >= 1 && 2 * K <= p.nz - 2;   // L u lives on interior planes only
#pragma unroll
        for (int s = 0; s < RC; ++s) {
            const T az = T(0.25) * hz2 * A[s];
            accB[s] += az;
            accA[s] += az;
            accC[s] += (zin ? T(0.5) * Q[s] + T(0.5) * a2 * A[s] : T(0)) - T(0.5) * hz2 * A[s];
        }
        // the coarse plane behind the walk is complete
        const int Kd = K - d;
        if (Kd >= Kb && Kd < Ke) {
#pragma unroll
            for (int s = 0; s < RC; ++s) {
                const int J = J0 + s;
                if (I > 0 && J < p.csy) rc[I + (long long)p.csx * J + p.csp * Kd] = -accB[s];
            }
        }
        if (K == K_last) break;
        // odd fine plane between K and K+d: weight 1/4 for both
        next_plane(2 * K + d, A, Q);
#pragma unroll
        for (int s = 0; s < RC; ++s) {
            const T v = T(0.25) * Q[s] + T(0.25) * a2 * A[s];
            accC[s] += v;
            accA[s] += v;
        }
#pragma unroll
        for (int s = 0; s < RC; ++s) {
            accB[s] = accC[s];
            accC[s] = accA[s];
            accA[s] = T(0);
        }
    }
}

template <typename T>
bool rr_launch(mhs_ctx* c, const Level& f, const void* u, const Level& co, void* rc, int down, const int* done, long long norm_n)
{
    constexpr int RC = RR_RC;
    const int ncx = f.sx / 2;
    if (f.sx % 2 || co.sx * 2 != f.sx || ncx < 8 || ncx > 512 || ((size_t)f.sx * sizeof(T)) % 16) return false;
    int G = std::max(1, MHS_RR_NT / ncx);
    while (G > 1 && RC * G > co.sy - 1) G >>= 1;                       // no more rows than the level has
    const size_t limit = 227 * 1024 - 1024;
    int nring = 0;
    for (; G >= 1; G >>= 1) {
        const size_t slot = (size_t)(2 * RC * G + 3) * f.sx * sizeof(T);
        nring = (int)std::min<size_t>(RR_MAXRING, (limit - 128) / slot);
        if (nring >= std::min(3, RR_MAXRING)) break;
    }
    if (G < 1 || nring < std::min(3, RR_MAXRING)) return false;
    auto kern = k_resid_restrict_ring<T>;
    static PerDevice attr;
    per_device(attr, c, [&] {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)limit);
        return 1;
    });
    RRP<T> p;
    p.sx = f.sx; p.sy = f.sy; p.nz = f.nz; p.sp = f.sp;
    p.tab = (const T*)f.tab;
    p.hz2 = (T)(1.0 / (f.hz * f.hz));
    p.a2 = (T)(c->alpha * c->alpha);
    p.csx = co.sx; p.csy = co.sy; p.cnz = co.nz; p.csp = co.sp;
    p.G = G;
    p.nring = nring;
    p.ntiles = (co.sy - 1 + RC * G - 1) / (RC * G);
    const int planes = co.nz - 2;
    // z-chunks: one CTA per SM, no chunk shorter than 4 coarse planes (2 n + 3 fine planes are read for n)
    p.nzc = std::max(1, std::min(planes / 4 > 0 ? planes / 4 : 1, c->num_sms * MHS_RR_CPS / p.ntiles));
    p.down = down;
    p.norm_partial = c->partial; p.norm_n = norm_n; p.ctl = c->ctl;
    if (norm_n > 0 && ((ncx * G) % 32 || !done)) return false;         // (the folded reduction works on whole warps)
    const size_t smem = 128 + (size_t)nring * (2 * RC * G + 3) * f.sx * sizeof(T) + 16;   // (+ the element after the last row)
    launch_pdl(c, kern, dim3((unsigned)(p.ntiles * p.nzc)), dim3((unsigned)(ncx * G)), smem, p, (const T*)u, (T*)rc, done);
    return true;
}

}  // namespace

// rhs_c <- R (0 - L u) on a level without a right-hand side (the finest 3D level); false: not launched (shape not
// supported), the caller takes k_resid_restrict_sep.
bool launch_resid_restrict_ring(mhs_ctx* c, const Level& f, const void* u, const Level& co, void* rc, int down, const int* done, long long norm_n)
{
    if (f.dim != 3 || f.nz < 5) return false;
    const bool ok = c->es == 8 ? rr_launch<double>(c, f, u, co, rc, down, done, norm_n) : rr_launch<float>(c, f, u, co, rc, down, done, norm_n);
    if (ok) { count_launch(c); c->prof.ring_restrict += 1; }
    return ok;
}

}  // namespace mhs
