// Field recovery as a bulk-copy fed streaming kernel (a8 + a9; eqs 9-10; readings C13-C15).
//
// Same formulas, in the same order, as k_fields_z / k_fields_ref (mhs_kernels_fields.cu):
//   Bz = -(dxx + dyy) P,  Bx = alpha D_y P + D_x D_z P,  By = -alpha D_x P + D_y D_z P,
//   p = p_b - xi Bz^2/(2 mu0),  rho = rho_b + (1/g) [ xi' Bz^2/(2 mu0) + (xi/mu0) B . grad Bz ]
// One pass: P is read once, the five outputs are written once (6w bytes per node).  k_fields_z kept the z-columns of P and
// of Bz in registers (126 of them), loaded through the L1 and stored 16-byte-strided 8-byte elements into the dense (odd
// pitch) outputs: 308 us at 257^3, 2.6 TB/s, latency-bound at 24 % occupancy.  Here a CTA owns a strip of R rows x all
// columns and a z-chunk; the R + 4 rows of P under it are one contiguous chunk of each plane in the aliased layout and come
// in through cp.async.bulk into a ring of planes, Bz of each plane is formed ONCE into a second ring (the density needs it at
// all six neighbours), one thread owns one column -- every shared-memory access is lane-contiguous, every global store is a
// run of consecutive 8-byte (4-byte) elements -- and no plane lives in registers.
// Step k:  Bz(k+2) from P(k+2)  |  outputs(k) from P(k-1..k+1), Bz(k-1..k+1)  |  one __syncthreads.
// The planes k = 0 (one-sided z differences, C13) and k = nz-1 (all wall) are left to the reference kernel.
#include <algorithm>
#include <cstdint>

#include "mhs_device.cuh"

namespace mhs {

namespace {

__device__ __forceinline__ uint32_t fr_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fr_bar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fr_smem(bar)), "r"(count));
}
__device__ __forceinline__ void fr_expect(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fr_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fr_bulk(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(fr_smem(dst)), "l"(src),
                 "r"(bytes), "r"(fr_smem(bar))
                 : "memory");
}
__device__ __forceinline__ void fr_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "FR_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra FR_DONE;\n"
        "bra FR_WAIT;\n"
        "FR_DONE:\n"
        "}\n" ::"r"(fr_smem(bar)),
        "r"(parity)
        : "memory");
}

constexpr int FR_NP = 5;   // ring of P planes: k-1 .. k+2 in use in step k, one more in flight
constexpr int FR_NB = 4;   // ring of Bz planes: k-1 .. k+2
constexpr int FR_NRO = 4;  // most output rows of one thread (rows of a strip / thread groups, rounded up)
constexpr int FR_NRB = 5;  // most Bz rows of one thread

template <typename T>
struct FRP {
    int nx, ny, nz, sx, sy;
    long long sp;
    T alpha, i2hx, i2hy, i2hz, ihx2, ihy2, i2mu0, imu0, ig;
    const T* ft;   // xi[nz] | dxi[nz] | p_b[nz] | rho_b[nz]
    int R, G;      // rows of a strip, thread groups along y (threads = sx * G)
    int nstrips, nzc;
};

// SX: row pitch (compile time: every shared-memory neighbour offset is an immediate), G: thread groups along y.
template <typename T, int SX, int G>
__global__ void __launch_bounds__(SX * G, 1) k_fields_ring(const __grid_constant__ FRP<T> q, const T* __restrict__ P, T* __restrict__ Bx,
                                                             T* __restrict__ By, T* __restrict__ Bzo, T* __restrict__ pp, T* __restrict__ rho)
{
    extern __shared__ __align__(128) unsigned char fsm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(fsm);
    const int R = q.R;
    const int pslot = (R + 4) * SX;                          // elements of a P slot: rows j0-2 .. j0+R+1
    const int bslot = (R + 2) * SX + 2;                      // elements of a Bz slot: rows j0-1 .. j0+R (+ pad)
    T* PR = reinterpret_cast<T*>(fsm + 128);
    T* BR = PR + FR_NP * pslot;
    const int i = (int)threadIdx.x % SX, g = (int)threadIdx.x / SX;
    const int strip = (int)blockIdx.x % q.nstrips, zc = (int)blockIdx.x / q.nstrips;
    const int j0 = 1 + strip * R;                            // first row of the strip (rows 1 .. sy-1 are interior)
    const int planes = q.nz - 2;
    const int kb = 1 + (int)((long long)planes * zc / q.nzc), ke = 1 + (int)((long long)planes * (zc + 1) / q.nzc);   // output planes [kb, ke)
    if (kb >= ke) return;
    const uint32_t pbytes = (uint32_t)pslot * (uint32_t)sizeof(T);
    const T* src0 = P + (long long)SX * (j0 - 2);            // (row j0-2, column 0) of plane 0

    if (threadIdx.x == 0) {
        for (int s = 0; s < FR_NP; ++s) fr_bar_init(bars + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // plane numbers are relative to kb-1: plane n = kb-1+n goes to P slot n % NP and Bz slot n % NB
    const int nload = ke - kb + 2;                           // planes kb-1 .. ke
    auto issue = [&](int n) {
        const int s = n % FR_NP;
        fr_expect(bars + s, pbytes);
        fr_bulk(PR + s * pslot, src0 + q.sp * (kb - 1 + n), pbytes, bars + s);
    };
    if (threadIdx.x == 0)
        for (int n = 0; n < min(FR_NP, nload); ++n) issue(n);

    const bool col_wall = i == 0;
    const int rows_b = min(R + 2, q.sy + 1 - (j0 - 1));      // Bz rows that exist (grid rows j0-1 .. sy)
    const int rows_o = min(R, q.sy - j0);                    // output rows (grid rows j0 .. sy-1)
    // Bz of plane n (relative) for this thread's share of the rows j0-1 .. j0+R, into its Bz slot; 0 on walls and on the top plane
    // (a thread group owns a run of CONSECUTIVE rows and walks along it with the rows j-1, j, j+1 of its column in registers)
    const int nrb = (rows_b + G - 1) / G, rb0 = g * nrb, rb1 = min(rows_b, rb0 + nrb);
    auto make_bz = [&](int n) {
        const int k = kb - 1 + n;
        const T* c = PR + (n % FR_NP) * pslot + (rb0 + 1) * SX + i;   // P slot row of grid row j0-1+r is r + 1
        T* bz = BR + (n % FR_NB) * bslot + rb0 * SX + i;
        const bool dead = k >= q.nz - 1 || col_wall;
        if (rb0 >= rb1) return;
        T vs = c[-SX], vc = c[0];
#pragma unroll
        for (int rr = 0; rr < FR_NRB; ++rr, c += SX, bz += SX) {     // (unrolled: the row window shifts by renaming)
            const int r = rb0 + rr;
            if (r >= rb1) break;
            const int j = j0 - 1 + r;
            const T vn = c[SX];
            T v = T(0);
            if (!(dead || j <= 0 || j >= q.sy)) {
                const T dxx = (c[1] - T(2) * vc + c[-1]) * q.ihx2;
                const T dyy = (vn - T(2) * vc + vs) * q.ihy2;
                v = -(dxx + dyy);
            }
            *bz = v;
            vs = vc; vc = vn;
        }
    };

    // warm-up: Bz of the planes kb-1, kb, kb+1
    for (int n = 0; n < min(3, nload); ++n) {
        fr_wait(bars + n % FR_NP, (uint32_t)((n / FR_NP) & 1));
        make_bz(n);
    }
    __syncthreads();

    const long long plane_d = (long long)q.nx * q.ny;
    const int nro = (rows_o + G - 1) / G, ro0 = g * nro, ro1 = min(rows_o, ro0 + nro);   // this group's output rows
    for (int k = kb; k < ke; ++k) {
        const int n = k - (kb - 1);                          // relative number of plane k
        // ---- Bz of plane k+2 ----
        if (n + 2 < nload) {
            fr_wait(bars + (n + 2) % FR_NP, (uint32_t)(((n + 2) / FR_NP) & 1));
            make_bz(n + 2);
        }
        // ---- outputs of plane k ----
        const int po0 = (ro0 + 2) * SX + i, bo0 = (ro0 + 1) * SX + i;
        const T* Pm = PR + ((n - 1) % FR_NP) * pslot + po0;
        const T* Pc = PR + (n % FR_NP) * pslot + po0;
        const T* Pp = PR + ((n + 1) % FR_NP) * pslot + po0;
        const T* Bm = BR + ((n - 1) % FR_NB) * bslot + bo0;
        const T* Bc = BR + (n % FR_NB) * bslot + bo0;
        const T* Bp = BR + ((n + 1) % FR_NB) * bslot + bo0;
        const T xi = q.ft[k], dxi = q.ft[q.nz + k], pb = q.ft[2 * q.nz + k], rb = q.ft[3 * q.nz + k];
        const T xi_mu = q.imu0 * xi;
        long long d = i + (long long)q.nx * (j0 + ro0) + plane_d * k;
        // the column's values on the rows j-1, j (s, c) of P(k-1), P(k), P(k+1), Bz(k); row j+1 (n) is loaded in the loop
        T pm_s = T(0), pm_c = T(0), pc_s = T(0), pc_c = T(0), pp_s = T(0), pp_c = T(0), bc_s = T(0), bc_c = T(0);
        if (ro0 < ro1) {
            pm_s = Pm[-SX]; pm_c = Pm[0]; pc_s = Pc[-SX]; pc_c = Pc[0]; pp_s = Pp[-SX]; pp_c = Pp[0]; bc_s = Bc[-SX]; bc_c = Bc[0];
        }
#pragma unroll
        for (int rr = 0; rr < FR_NRO; ++rr, Pm += SX, Pc += SX, Pp += SX, Bm += SX, Bc += SX, Bp += SX, d += q.nx) {
            if (ro0 + rr >= ro1) break;
            const T pm_n = Pm[SX], pc_n = Pc[SX], pp_n = Pp[SX], bc_n = Bc[SX];
            T bx = T(0), by = T(0), bz = T(0), pv = pb, rv = rb;
            if (!col_wall) {
                bz = bc_c;
                const T dzn = (pp_n - pm_n) * q.i2hz, dzs = (pp_s - pm_s) * q.i2hz;
                const T dzR = (Pp[1] - Pm[1]) * q.i2hz, dzL = (Pp[-1] - Pm[-1]) * q.i2hz;
                bx = q.alpha * (pc_n - pc_s) * q.i2hy + (dzR - dzL) * q.i2hx;
                by = -q.alpha * (Pc[1] - Pc[-1]) * q.i2hx + (dzn - dzs) * q.i2hy;
                const T dxBz = (Bc[1] - Bc[-1]) * q.i2hx;
                const T dyBz = (bc_n - bc_s) * q.i2hy;
                const T dzBz = (Bp[0] - Bm[0]) * q.i2hz;
                pv = pb - xi * bz * bz * q.i2mu0;
                rv = rb + q.ig * (dxi * bz * bz * q.i2mu0 + xi_mu * (bx * dxBz + by * dyBz + bz * dzBz));
            }
            if (Bx) { Bx[d] = bx; By[d] = by; Bzo[d] = bz; }
            if (pp) pp[d] = pv;
            if (rho) rho[d] = rv;
            if (col_wall) {   // the aliased wall node (nx-1, j)
                const long long dw = d + q.nx - 1;
                if (Bx) { Bx[dw] = T(0); By[dw] = T(0); Bzo[dw] = T(0); }
                if (pp) pp[dw] = pb;
                if (rho) rho[dw] = rb;
            }
            pm_s = pm_c; pm_c = pm_n; pc_s = pc_c; pc_c = pc_n; pp_s = pp_c; pp_c = pp_n; bc_s = bc_c; bc_c = bc_n;
        }
        // the wall rows j = 0 (first strip) and j = ny-1 (last strip): B = 0, background p and rho
        if (g == 0 && (strip == 0 || strip == q.nstrips - 1)) {
            for (int e = 0; e < 2; ++e) {
                if ((e == 0 && strip != 0) || (e == 1 && strip != q.nstrips - 1)) continue;
                const int j = e == 0 ? 0 : q.ny - 1;
                const long long dd = i + (long long)q.nx * j + plane_d * k;
                if (Bx) { Bx[dd] = T(0); By[dd] = T(0); Bzo[dd] = T(0); }
                if (pp) pp[dd] = pb;
                if (rho) rho[dd] = rb;
                if (col_wall) {
                    const long long dw = dd + q.nx - 1;
                    if (Bx) { Bx[dw] = T(0); By[dw] = T(0); Bzo[dw] = T(0); }
                    if (pp) pp[dw] = pb;
                    if (rho) rho[dw] = rb;
                }
            }
        }
        __syncthreads();      // Bz(k+2) complete; P(k-1) and Bz(k-1) no longer needed
        if (threadIdx.x == 0 && n - 1 + FR_NP < nload) issue(n - 1 + FR_NP);
    }
}

template <typename T>
bool fr_launch(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho)
{
    const int sx = lv.sx;
    if (!(sx == 32 || sx == 64 || sx == 128 || sx == 256 || sx == 512 || sx == 1024) || lv.sy < 8 || lv.nz < 5) return false;
    const int G = std::max(1, 512 / sx);
    const size_t limit = 227 * 1024 - 1024;
    // rows per strip (<= 8, as many as the shared memory takes) and z-chunks: the pair that keeps the SMs busiest over whole
    // waves of CTAs (one CTA per SM: the rings take most of the shared memory), then the one with the least halo
    int best = 0, best_nzc = 1;
    double bscore = -1.0;
    for (int R = 2; R <= 8; ++R) {
        const size_t smem = 128 + ((size_t)FR_NP * (R + 4) * sx + (size_t)FR_NB * ((R + 2) * sx + 2)) * sizeof(T);
        if (smem > limit) break;
        if ((R + G - 1) / G > FR_NRO || (R + 2 + G - 1) / G > FR_NRB) break;
        const int ns = (lv.sy - 1 + R - 1) / R;
        const int maxc = std::max(1, (lv.nz - 2) / 16);
        for (int nzc = 1; nzc <= maxc; ++nzc) {
            const long long ctas = (long long)ns * nzc;
            const long long waves = (ctas + c->num_sms - 1) / c->num_sms;
            const double eff = (double)ctas / (double)(waves * c->num_sms);
            const double len = (double)(lv.nz - 2) / nzc;
            const double score = eff * (R / (R + 4.0) + 0.2) * (len / (len + 3.0));    // 3 warm-up planes per chunk
            if (score > bscore + 1e-9) { bscore = score; best = R; best_nzc = nzc; }
        }
    }
    if (!best) return false;
    FRP<T> q;
    q.nx = lv.nx; q.ny = lv.ny; q.nz = lv.nz; q.sx = lv.sx; q.sy = lv.sy; q.sp = lv.sp;
    q.alpha = (T)c->alpha;
    q.i2hx = (T)(1.0 / (2.0 * lv.hx)); q.i2hy = (T)(1.0 / (2.0 * lv.hy)); q.i2hz = (T)(1.0 / (2.0 * lv.hz));
    q.ihx2 = (T)(1.0 / (lv.hx * lv.hx)); q.ihy2 = (T)(1.0 / (lv.hy * lv.hy));
    q.i2mu0 = (T)(1.0 / (2.0 * c->opt.mu0)); q.imu0 = (T)(1.0 / c->opt.mu0); q.ig = (T)(1.0 / c->opt.g);
    q.ft = (const T*)c->prof_tab;
    q.R = best; q.G = G;
    q.nstrips = (lv.sy - 1 + best - 1) / best;
    q.nzc = best_nzc;
    const size_t smem = 128 + ((size_t)FR_NP * (best + 4) * sx + (size_t)FR_NB * ((best + 2) * sx + 2)) * sizeof(T);
    const long long N = lv.npts();
    T* Bp = (T*)B;
    const dim3 grid((unsigned)(q.nstrips * q.nzc));
#define FR_GO(SXV, GV)                                                                                                              \
    do {                                                                                                                            \
        auto kern = k_fields_ring<T, SXV, GV>;                                                                                      \
        static PerDevice attr;                                                                                                      \
        per_device(attr, c, [&] {                                                                                                   \
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)limit);                                    \
            return 1;                                                                                                               \
        });                                                                                                                         \
        kern<<<grid, dim3(SXV * GV), smem, c->stream>>>(q, (const T*)P, Bp, Bp ? Bp + N : nullptr, Bp ? Bp + 2 * N : nullptr, (T*)p, \
                                                        (T*)rho);                                                                   \
        return true;                                                                                                                \
    } while (0)
    switch (sx) {
        case 32: FR_GO(32, 16);
        case 64: FR_GO(64, 8);
        case 128: FR_GO(128, 4);
        case 256: FR_GO(256, 2);
        case 512: FR_GO(512, 1);
        case 1024: FR_GO(1024, 1);
        default: break;
    }
#undef FR_GO
    return false;
}

}  // namespace

// planes 1 .. nz-2 of B, p, rho; false: shape not supported (the caller takes k_fields_z)
bool launch_fields_ring(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho)
{
    if (lv.dim != 3) return false;
    const bool ok = c->es == 8 ? fr_launch<double>(c, lv, P, B, p, rho) : fr_launch<float>(c, lv, P, B, p, rho);
    if (ok) count_launch(c);
    return ok;
}

}  // namespace mhs
