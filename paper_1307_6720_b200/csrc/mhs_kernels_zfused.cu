// Temporally blocked weighted-Jacobi smoother of libmhs_b200 for sm_100a: S sweeps (a2) in ONE
// pass over HBM -- the iterate is read once and written once whatever S is (2w/S bytes per update).
//
// Scheme ("bulk-copy fed z-streaming pipeline"):
//   * The aliased Dirichlet layout (mhs_internal.h) makes a tile of full rows of one plane ONE contiguous chunk
//     of memory, so the input planes are brought in by the bulk-copy engine (cp.async.bulk global -> shared,
//     completion on an mbarrier: the TMA data path without a tensor map) into a ring of NIN planes, several
//     planes ahead of the arithmetic; no register or thread is spent on prefetching.
//   * A CTA owns a tile of WY*R rows x TC columns and walks up in z.  Stage s of the pipeline lags one plane
//     behind stage s-1: at step t stage 1 makes sweep-1 values of plane t-1 from the input planes t-2, t-1, t,
//     stage 2 makes sweep-2 values of plane t-2 from sweep-1 planes t-3, t-2, t-1, ...  A thread keeps the z-column
//     (below, centre) of its R x V nodes of every stage in registers; in-plane neighbours come from registers
//     (rows of its own strip), warp shuffles (x) and a single shared-memory copy of the stage's centre plane.
//   * Every stage shrinks the valid region by one row/plane at tile and chunk edges: a tile makes WY*R-2(S-1)
//     output rows, a z-segment is warmed up over S planes.  Walls are held fixed in every stage; the bottom
//     (data) and top planes pass through every stage by coefficients (A = 1, B = 0), so no branch is needed.
//   * fp64 uses the expanded update  u' = (1-w) u + Bx (e+w) + By (n+s) + Bz (up+dn) + W f  with per-plane
//     Bx = -(w/D) c/hx^2 ... : 7-8 DP instructions per update instead of 13 -- with S sweeps per byte the DP
//     pipe (64 lanes/clk/SM), not HBM, would otherwise set the pace.  fp32 keeps the difference form (C20).
//   * The squared norm of the residual of the INPUT iterate is a by-product of stage 1 (r = (u'-u) D/w).
//   * Work is a linearised list of (tile, plane) pairs cut into equal contiguous ranges, one per CTA, one CTA
//     per SM: no wave quantisation whatever the grid size.
#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "mhs_device.cuh"

namespace mhs {

template <typename T> struct ZV;
template <> struct ZV<double> { static constexpr int N = 2; };
template <> struct ZV<float> { static constexpr int N = 4; };

template <typename T>
struct __align__(16) ZVec {
    T v[ZV<T>::N];
};

template <typename T>
struct ZP {
    int sx, sy, nz;
    long long sp;
    const T* tab;       // 10*nz: cx|cy|diag|w | A|Bx|By|Bz|iw|wz   (mhs_api.cu build_hierarchy)
    T cz, a2;
    int WX, WY;         // warps per tile along x / y
    int TC, COUT, ntx;  // tile columns, output columns per tile, tiles along x (1: the tile is a full row)
    int ROUT, nty;      // output rows per tile, tiles along y
    int NP;             // interior planes nz-2
    long long items;    // ntx*nty*NP
    int nin;            // input ring depth
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "ZW_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra ZW_DONE;\n"
        "bra ZW_WAIT;\n"
        "ZW_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ double zshfl_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float zshfl_up(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double zshfl_dn(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float zshfl_dn(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename T>
struct Coef {   // per-plane coefficients of one sweep
    T cx, cy, A, Bx, By, Bz, iw, wz;
};

template <typename T>
__device__ __forceinline__ Coef<T> coef_at(const ZP<T>& p, int k)
{
    k = min(max(k, 0), p.nz - 1);
    Coef<T> c;
    const T* t = p.tab;
    c.cx = t[k]; c.cy = t[p.nz + k];
    c.A = t[4 * p.nz + k]; c.Bx = t[5 * p.nz + k]; c.By = t[6 * p.nz + k]; c.Bz = t[7 * p.nz + k];
    c.iw = t[8 * p.nz + k]; c.wz = t[9 * p.nz + k];
    return c;
}

// One Jacobi update of the V nodes of a vector.  c: centre values, cw/ce: the nodes left/right of the vector,
// n/s: the rows above/below, up/dn: the planes above/below, f: right-hand side.  The fp32 version also returns
// res = rhs - L u; in fp64 the caller recovers it from (out - c) * iw.
template <bool HAS_RHS>
__device__ __forceinline__ void jacobi_vec_d(const Coef<double>& k, const ZVec<double>& c, double cw, double ce, const ZVec<double>& n,
                                             const ZVec<double>& s, const ZVec<double>& up, const ZVec<double>& dn, const ZVec<double>& f,
                                             ZVec<double>& out)
{
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const double w = e == 0 ? cw : c.v[0];
        const double ea = e == 1 ? ce : c.v[1];
        double o = k.A * c.v[e];
        o = fma(k.Bx, ea + w, o);
        o = fma(k.By, n.v[e] + s.v[e], o);
        o = fma(k.Bz, up.v[e] + dn.v[e], o);
        if (HAS_RHS) o = fma(k.wz, f.v[e], o);
        out.v[e] = o;
    }
}

template <bool HAS_RHS>
__device__ __forceinline__ void jacobi_vec_f(const Coef<float>& k, float cz, float a2, const ZVec<float>& c, float cw, float ce,
                                             const ZVec<float>& n, const ZVec<float>& s, const ZVec<float>& up, const ZVec<float>& dn,
                                             const ZVec<float>& f, ZVec<float>& out, ZVec<float>& res)
{
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const float w = e == 0 ? cw : c.v[e - 1];
        const float ea = e == 3 ? ce : c.v[e + 1];
        float lu = k.cx * lap1<float>(ea, w, c.v[e]) + k.cy * lap1<float>(n.v[e], s.v[e], c.v[e]);
        lu += cz * lap1<float>(up.v[e], dn.v[e], c.v[e]) + a2 * c.v[e];
        const float r = (HAS_RHS ? f.v[e] : 0.f) - lu;
        res.v[e] = r;
        out.v[e] = c.v[e] + k.wz * r;
    }
}

template <typename T>
__device__ __forceinline__ ZVec<T> zld(const T* p) { return *reinterpret_cast<const ZVec<T>*>(p); }
template <typename T>
__device__ __forceinline__ void zst(T* p, const ZVec<T>& a) { *reinterpret_cast<ZVec<T>*>(p) = a; }

// ------------------------------------------------------------------------------------------------
// S sweeps.  ZERO: the input iterate is identically zero (coarse-grid correction, first pre-sweep):
// sweep 1 is u = (omega/D) rhs and no input plane is read at all.
// ------------------------------------------------------------------------------------------------
template <typename T, int S, bool HAS_RHS, bool ZERO, bool NORM>
__global__ void __launch_bounds__(512, 1) k_zsweep(const __grid_constant__ ZP<T> p, const T* __restrict__ u, const T* __restrict__ rhs,
                                                    T* __restrict__ out, double* __restrict__ partial, const int* __restrict__ done)
{
    static_assert(S == 1 || S == 2, "S sweeps per pass: 1 or 2");
    static_assert(!ZERO || HAS_RHS, "a zero iterate with a zero right-hand side stays zero");
    if (done && *done) return;
    constexpr int V = ZV<T>::N;
    constexpr int R = 4;
    extern __shared__ __align__(128) unsigned char zsm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wx = warp % p.WX, wy = warp / p.WX;
    const int TC = p.TC;
    const int rows_in = p.WY * R + 2;                       // input tile: one halo row below and above
    const int in_plane = rows_in * TC;                      // elements
    // shared memory: [mbarriers: 8 x 8 B, padded to 128] [IN ring: nin planes] [EX: (WY*R + 2) rows, guard row each side]
    uint64_t* bars = reinterpret_cast<uint64_t*>(zsm);
    T* IN = reinterpret_cast<T*>(zsm + 128);
    T* EX = IN + (size_t)(ZERO ? 0 : p.nin) * in_plane + TC;   // -> row 0 of the exchange tile (guard row before it)

    if (!ZERO && threadIdx.x == 0) {
        for (int q = 0; q < p.nin; ++q) mbar_init(bars + q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int cx0 = (wx * 32 + lane) * V;                   // first column of this thread's vector inside the tile
    const long long q0 = p.items * blockIdx.x / gridDim.x, q1 = p.items * (blockIdx.x + 1) / gridDim.x;
    int nload = 0;                                          // planes requested so far by this CTA (ring position)
    int nwait = 0;                                          // planes consumed so far
    double acc = 0.0;

    for (long long q = q0; q < q1;) {
        const int tile = (int)(q / p.NP);
        const int kb = 1 + (int)(q - (long long)tile * p.NP);
        const int ke = (int)min((long long)p.NP + 1, kb + (q1 - q));   // output planes [kb, ke)
        q += ke - kb;
        const int ty = tile / p.ntx, tx = tile - ty * p.ntx;
        const int ct = p.ntx == 1 ? 0 : tx * p.COUT - V;              // first column of the tile
        const int jt = ty * p.ROUT - (S - 1);                          // first row of the strips
        const int kstart = max(kb - S, 0), kend_in = min(ke - 1 + S, p.nz - 1);
        const T* tile_src = u + (long long)(jt - 1) * p.sx + ct;      // (row jt-1, col ct) of plane 0
        const uint32_t plane_bytes = (uint32_t)in_plane * sizeof(T);

        auto issue = [&](int k) {   // warp 0: request input plane k into ring slot nload % nin
            const int slot = nload % p.nin;
            T* dst = IN + (size_t)slot * in_plane;
            const T* src = tile_src + p.sp * k;
            if (lane == 0) mbar_expect_tx(bars + slot, plane_bytes);
            __syncwarp();
            if (p.ntx == 1) {
                if (lane == 0) bulk_g2s(dst, src, plane_bytes, bars + slot);
            } else {
                for (int r = lane; r < rows_in; r += 32) bulk_g2s(dst + r * TC, src + (long long)r * p.sx, (uint32_t)(TC * sizeof(T)), bars + slot);
            }
        };
        int knext = kstart;     // next plane to request
        if (!ZERO) {
            if (warp == 0)
                for (int n = 0; n < p.nin && knext + n <= kend_in; ++n) { issue(knext + n); ++nload; }
            else
                nload += min(p.nin, kend_in - knext + 1);
            knext += min(p.nin, kend_in - knext + 1);
        }

        // wall / validity masks of this thread's nodes
        const int jrow0 = jt + wy * R;                                  // grid row of strip row 0
        const int icol0 = ct + cx0;                                     // grid column of vector element 0
        bool colwall[V];
#pragma unroll
        for (int e = 0; e < V; ++e) colwall[e] = (icol0 + e == 0) || (icol0 + e == p.sx);
        const bool col_out = p.ntx == 1 ? true : (cx0 >= V && cx0 < TC - V && icol0 < p.sx);
        bool rowwall[R], row_out[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int j = jrow0 + r;
            rowwall[r] = (j == 0) || (j == p.sy);
            const int jo = j - ty * p.ROUT;
            row_out[r] = jo >= 0 && jo < p.ROUT && j > 0 && j < p.sy;
        }

        ZVec<T> cm0[R], cc0[R], cm1[R], cc1[R], fprev[R];
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int e = 0; e < V; ++e) { cm0[r].v[e] = cc0[r].v[e] = cm1[r].v[e] = cc1[r].v[e] = fprev[r].v[e] = T(0); }

        const long long own = (long long)jrow0 * p.sx + icol0;          // in-plane offset of (strip row 0, element 0)

        for (int t = kstart; t <= ke - 1 + S; ++t) {
            // ---------------- stage 1: sweep-1 values of plane t-1 ----------------
            const int p1 = t - 1;
            const bool act1 = p1 >= kstart && p1 <= kend_in;
            ZVec<T> cp0[R], u1[R], f1[R];
            if (!ZERO) {
                if (t <= kend_in) {
                    const int slot = nwait % p.nin;
                    mbar_wait(bars + slot, (uint32_t)((nwait / p.nin) & 1));
                    const T* pin = IN + (size_t)slot * in_plane + (wy * R + 1) * TC + cx0;
#pragma unroll
                    for (int r = 0; r < R; ++r) cp0[r] = zld(pin + r * TC);
                } else {
#pragma unroll
                    for (int r = 0; r < R; ++r)
#pragma unroll
                        for (int e = 0; e < V; ++e) cp0[r].v[e] = T(0);
                }
            }
            if (HAS_RHS && act1) {
#pragma unroll
                for (int r = 0; r < R; ++r) f1[r] = zld(rhs + own + p.sp * p1 + (long long)r * p.sx);
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int e = 0; e < V; ++e) f1[r].v[e] = T(0);
            }
            if (ZERO) {
                const Coef<T> k1 = coef_at(p, p1);
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int e = 0; e < V; ++e) u1[r].v[e] = (rowwall[r] || colwall[e] || !act1) ? T(0) : k1.wz * f1[r].v[e];
            } else if (act1) {
                const Coef<T> k1 = coef_at(p, p1);
                // centre plane t-1 sits in the ring slot requested just before the current one
                const int slotc = (nwait - 1 + p.nin) % p.nin;
                const T* pc = IN + (size_t)slotc * in_plane + (wy * R + 1) * TC + cx0;
                const ZVec<T> sbot = zld(pc - TC);
                const ZVec<T> ntop = zld(pc + R * TC);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    T cw = zshfl_up(cc0[r].v[V - 1]);
                    T ce = zshfl_dn(cc0[r].v[0]);
                    if (lane == 0) cw = pc[r * TC - 1];
                    if (lane == 31) ce = pc[r * TC + V];
                    ZVec<T> o, res;
                    const ZVec<T>& nn = r == R - 1 ? ntop : cc0[r + 1 < R ? r + 1 : r];
                    const ZVec<T>& ss = r == 0 ? sbot : cc0[r > 0 ? r - 1 : 0];
                    if constexpr (sizeof(T) == 8) {
                        jacobi_vec_d<HAS_RHS>(k1, cc0[r], cw, ce, nn, ss, cp0[r], cm0[r], f1[r], o);
                    } else {
                        jacobi_vec_f<HAS_RHS>(k1, p.cz, p.a2, cc0[r], cw, ce, nn, ss, cp0[r], cm0[r], f1[r], o, res);
                    }
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const bool wall = rowwall[r] || colwall[e];
                        if (NORM && !wall && row_out[r] && col_out && p1 >= kb && p1 < ke) {
                            double rr;
                            if constexpr (sizeof(T) == 8) rr = (o.v[e] - cc0[r].v[e]) * k1.iw;
                            else rr = (double)res.v[e];
                            acc += rr * rr;
                        }
                        u1[r].v[e] = wall ? cc0[r].v[e] : o.v[e];
                    }
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) u1[r] = cc0[r];
            }

            if (S == 1) {
                if (p1 >= kb && p1 < ke && col_out) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if (row_out[r]) zst(out + own + p.sp * p1 + (long long)r * p.sx, u1[r]);
                }
            }

            // ---------------- stage 2: sweep-2 values of plane t-2 ----------------
            if (S == 2) {
                const int p2 = t - 2;
                if (p2 >= kstart && p2 <= kend_in) {
                    const Coef<T> k2 = coef_at(p, p2);
                    const T* pe = EX + (wy * R) * TC + cx0;             // exchange tile holds sweep-1 plane t-2
                    const ZVec<T> sbot = zld(pe - TC);
                    const ZVec<T> ntop = zld(pe + R * TC);
                    const bool st = p2 >= kb && p2 < ke && col_out;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        T cw = zshfl_up(cc1[r].v[V - 1]);
                        T ce = zshfl_dn(cc1[r].v[0]);
                        if (lane == 0) cw = pe[r * TC - 1];
                        if (lane == 31) ce = pe[r * TC + V];
                        ZVec<T> o, res;
                        const ZVec<T>& nn = r == R - 1 ? ntop : cc1[r + 1 < R ? r + 1 : r];
                        const ZVec<T>& ss = r == 0 ? sbot : cc1[r > 0 ? r - 1 : 0];
                        if constexpr (sizeof(T) == 8) {
                            jacobi_vec_d<HAS_RHS>(k2, cc1[r], cw, ce, nn, ss, u1[r], cm1[r], fprev[r], o);
                        } else {
                            jacobi_vec_f<HAS_RHS>(k2, p.cz, p.a2, cc1[r], cw, ce, nn, ss, u1[r], cm1[r], fprev[r], o, res);
                        }
#pragma unroll
                        for (int e = 0; e < V; ++e)
                            if (rowwall[r] || colwall[e]) o.v[e] = cc1[r].v[e];
                        if (st && row_out[r]) zst(out + own + p.sp * p2 + (long long)r * p.sx, o);
                    }
                }
            }

            __syncthreads();   // every read of the ring slot of plane t-1 and of the exchange tile is done
            if (!ZERO) {
                if (t <= kend_in) ++nwait;
                // the slot of plane t-1 is free: request the next plane into it
                if (t > kstart && knext <= kend_in) {
                    if (warp == 0) issue(knext);
                    ++nload; ++knext;
                }
            }
            if (S == 2) {
                T* pe = EX + (wy * R) * TC + cx0;
#pragma unroll
                for (int r = 0; r < R; ++r) zst(pe + r * TC, u1[r]);
                __syncthreads();   // sweep-1 plane t-1 is visible
#pragma unroll
                for (int r = 0; r < R; ++r) { cm1[r] = cc1[r]; cc1[r] = u1[r]; fprev[r] = f1[r]; }
            }
            if (!ZERO) {
#pragma unroll
                for (int r = 0; r < R; ++r) { cm0[r] = cc0[r]; cc0[r] = cp0[r]; }
            }
        }
        // drain: planes requested but not consumed cannot exist (requests stop at kend_in, steps run past it)
    }
    if (NORM) {
        __shared__ double s_red[16];
        acc = warp_sum(acc);
        if (lane == 0) s_red[warp] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double v = 0.0;
            for (int q = 0; q < (int)(blockDim.x >> 5); ++q) v += s_red[q];
            partial[blockIdx.x] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
struct ZCfg {
    bool ok = false;
    int WX = 0, WY = 4, TC = 0, COUT = 0, ntx = 1, ROUT = 0, nty = 0, nin = 4, ctas = 0;
    size_t smem = 0;
};

template <typename T>
static ZCfg zcfg(const mhs_ctx* c, const Level& lv, int S, bool zero)
{
    constexpr int V = ZV<T>::N;
    constexpr int R = 4;
    ZCfg z;
    if (lv.dim != 3 || lv.coarsest || lv.nz < 5 || lv.sy < 32) return z;
    const int lane_cols = 32 * V;
    if (lv.sx % lane_cols != 0) return z;
    const int wfull = lv.sx / lane_cols;
    z.WY = 4;
    if (wfull <= 4) {
        z.WX = wfull; z.ntx = 1; z.TC = lv.sx; z.COUT = lv.sx;
    } else {
        // x tiles with one halo vector per side: pick the width (3 or 4 warps) that wastes fewer columns
        int best = 0; double bw = 1e30;
        for (int w = 3; w <= 4; ++w) {
            const int cout = w * lane_cols - 2 * V;
            const int n = (lv.sx + cout - 1) / cout;
            const double waste = (double)n * w * lane_cols / lv.sx;
            if (waste < bw) { bw = waste; best = w; }
        }
        z.WX = best; z.TC = best * lane_cols; z.COUT = z.TC - 2 * V; z.ntx = (lv.sx + z.COUT - 1) / z.COUT;
    }
    z.ROUT = z.WY * R - 2 * (S - 1);
    z.nty = (lv.sy + z.ROUT - 1) / z.ROUT;
    const size_t in_plane = (size_t)(z.WY * R + 2) * z.TC * sizeof(T);
    const size_t ex = (size_t)(z.WY * R + 2) * z.TC * sizeof(T);
    z.nin = 4;
    while (z.nin > 2 && 128 + (zero ? 0 : z.nin * in_plane) + ex + 256 > 227 * 1024) --z.nin;
    z.smem = 128 + (zero ? 0 : z.nin * in_plane) + ex + 256;
    if (z.smem > 227 * 1024) return z;
    const long long items = (long long)z.ntx * z.nty * (lv.nz - 2);
    // one CTA per SM; a z-segment should be long against its S warm-up planes
    z.ctas = (int)std::max<long long>(1, std::min<long long>(c->num_sms, items / 12));
    z.ok = true;
    return z;
}

template <typename T, int S, bool HAS_RHS, bool ZERO, bool NORM>
static int zsweep_launch(mhs_ctx* c, const Level& lv, const ZCfg& z, const void* u, const void* rhs, void* out, const int* done)
{
    auto kern = k_zsweep<T, S, HAS_RHS, ZERO, NORM>;
    static bool attr = false;
    if (!attr) {
        cudaFuncAttributes fa;
        size_t stat = 4096;
        if (cudaFuncGetAttributes(&fa, kern) == cudaSuccess) stat = fa.sharedSizeBytes;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024 - stat));
        attr = true;
    }
    ZP<T> p;
    p.sx = lv.sx; p.sy = lv.sy; p.nz = lv.nz; p.sp = lv.sp;
    p.tab = (const T*)lv.tab;
    p.cz = (T)(1.0 / (lv.hz * lv.hz));
    p.a2 = (T)(c->alpha * c->alpha);
    p.WX = z.WX; p.WY = z.WY; p.TC = z.TC; p.COUT = z.COUT; p.ntx = z.ntx; p.ROUT = z.ROUT; p.nty = z.nty;
    p.NP = lv.nz - 2;
    p.items = (long long)z.ntx * z.nty * p.NP;
    p.nin = z.nin;
    kern<<<z.ctas, z.WX * z.WY * 32, z.smem, c->stream>>>(p, (const T*)u, (const T*)rhs, (T*)out, c->partial, done);
    if (getenv("MHS_DEBUG")) {
        cudaError_t e = cudaPeekAtLastError();
        fprintf(stderr, "[mhs] k_zsweep<%s,S=%d,rhs=%d,zero=%d,norm=%d> %dx%dx%d WX %d WY %d TC %d ntx %d nty %d nin %d ctas %d smem %zu: %s\n",
                sizeof(T) == 8 ? "f64" : "f32", S, (int)HAS_RHS, (int)ZERO, (int)NORM, lv.nx, lv.ny, lv.nz, z.WX, z.WY, z.TC, z.ntx, z.nty, z.nin,
                z.ctas, z.smem, cudaGetErrorString(e));
    }
    return z.ctas;
}

bool zsweep_ok(const mhs_ctx* c, const Level& lv)
{
    return c->es == 8 ? zcfg<double>(c, lv, 2, false).ok : zcfg<float>(c, lv, 2, false).ok;
}

// S (1 or 2) sweeps of level lv: u -> out.  zero: u is identically zero (not read).  norm: partial sums of the
// squared residual of u go to c->partial; returns their number (0 without norm).
int launch_zsweep(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int S, bool zero, bool norm, const int* done)
{
    count_launch(c);
#define ZS(T, SS, RHS, ZERO, NORM)                                                        \
    do {                                                                                  \
        const ZCfg z = zcfg<T>(c, lv, SS, ZERO);                                          \
        const int n = zsweep_launch<T, SS, RHS, ZERO, NORM>(c, lv, z, u, rhs, out, done); \
        return NORM ? n : 0;                                                              \
    } while (0)
#define ZT(T)                                             \
    do {                                                  \
        if (zero) {                                       \
            if (S == 2) ZS(T, 2, true, true, false);      \
            ZS(T, 1, true, true, false);                  \
        } else if (rhs) {                                 \
            if (S == 2) {                                 \
                if (norm) ZS(T, 2, true, false, true);    \
                ZS(T, 2, true, false, false);             \
            }                                             \
            if (norm) ZS(T, 1, true, false, true);        \
            ZS(T, 1, true, false, false);                 \
        } else {                                          \
            if (S == 2) {                                 \
                if (norm) ZS(T, 2, false, false, true);   \
                ZS(T, 2, false, false, false);            \
            }                                             \
            if (norm) ZS(T, 1, false, false, true);       \
            ZS(T, 1, false, false, false);                \
        }                                                 \
    } while (0)
    if (c->es == 8) ZT(double);
    else ZT(float);
#undef ZT
#undef ZS
    return 0;
}

}  // namespace mhs
