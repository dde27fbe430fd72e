// Temporally blocked weighted-Jacobi smoother of libmhs_b200 for sm_100a: S sweeps (a2) in ONE
// pass over HBM -- the iterate is read once and written once whatever S is (2w/S bytes per update).
//
// Scheme ("bulk-copy fed z-streaming pipeline"):
//   * The aliased Dirichlet layout (mhs_internal.h) makes a tile of full rows of one plane ONE contiguous chunk
//     of memory, so the input planes are brought in by the bulk-copy engine (cp.async.bulk global -> shared,
//     completion on an mbarrier: the TMA data path without a tensor map) into a ring of NIN planes, several
//     planes ahead of the arithmetic; no register or thread is spent on prefetching.
//   * "Few fat threads": a thread owns 8 rows x one vector (ZR = 8, 256 threads per CTA, up to 255 registers), and the
//     shared-memory operands of a row are fetched one row ahead of its arithmetic.  Measured at 257^3: 4 rows x 512 threads
//     x 128 registers 68 us per 2-sweep pass, the same with row-ahead loads 66 us (ptxas sinks the loads back to their uses
//     when registers are short), 8 rows x 256 threads x 254 registers 62.5 us -- latency is hidden by ILP, not by warps.
//   * A CTA owns a tile of ZWY*ZR rows x TC columns and walks up in z.  Stage s of the pipeline lags one plane
//     behind stage s-1: at step t stage 1 makes sweep-1 values of plane t-1 from the input planes t-2, t-1, t,
//     stage 2 makes sweep-2 values of plane t-2 from sweep-1 planes t-3, t-2, t-1.  A thread owns a patch of
//     8 (fp64) or 4 (fp32) rows x one 128-bit vector and keeps the z-column (below, centre, above) of its patch for
//     every stage in registers; steps come in pairs whose register sets swap roles by renaming.  In-plane neighbours: rows of its own patch from registers, everything else from shared memory --
//     the ring slot of the centre plane for stage 1, a double-buffered exchange plane for stage 2 -- with
//     plain LDS (no shuffles, no lane-dependent branches).  One __syncthreads per plane.
//   * Every stage shrinks the valid region by one row/plane at tile and chunk edges: a tile makes 16-2(S-1)
//     output rows, a z-segment is warmed up over S planes.  Walls are held fixed in every stage; the bottom
//     (data) and top planes pass through every stage by coefficients (A = 1, B = 0), so no branch is needed.
//   * fp64 uses the expanded update  u' = (1-w) u + Bx (e+w) + By (n+s) + Bz (up+dn) + W f  with per-plane
//     Bx = -(w/D) c/hx^2 ... : 7 DP instructions per update.  fp32 keeps the difference form (C20).
//   * The squared norm of the residual of the INPUT iterate is a by-product of stage 1 (r = (u'-u) D/w).
//   * Work is a linearised list of (tile, plane) pairs cut into equal contiguous ranges, one per CTA, one CTA
//     per SM: no wave quantisation whatever the grid size.
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <mutex>
#include <tuple>

#include "mhs_device.cuh"

namespace mhs {

template <typename T> struct ZV;
// N: elements of a 128-bit vector; NCO: coefficients per plane record; R: rows of a thread's patch; WY: warps of a tile
// along y (a tile has WY*R = 16 patch rows).  fp64: 8 rows x 256 threads x <= 255 registers ("few fat threads": measured
// 62.5 us per 2-sweep pass at 257^3 against 68 us for 4 rows x 512 threads); fp32, with half the registers per value and the
// longer difference-form update, is faster the other way round (1025^2 x 257: 632 us against 900 us per pass).
#ifndef MHS_ZR64
#define MHS_ZR64 8
#endif
template <> struct ZV<double> { static constexpr int N = 2, NCO = 6, R = MHS_ZR64, WY = 16 / MHS_ZR64; };
template <> struct ZV<float> { static constexpr int N = 4, NCO = 4, R = 4, WY = 4; };

// Tile geometry is a compile-time function of WXT (warps along x), so that every shared-memory stride is an immediate:
template <typename T, int WXT> struct ZG {
    static constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY;
    static constexpr int TC = WXT * 32 * ZV<T>::N;          // tile columns
    static constexpr int INP = (ZWY * ZR + 2) * TC;         // elements of one ring slot / exchange plane
    // prolongation-fused variant (full-row tiles only): the coarse rows under the ZWY*ZR+2 fine rows of a tile
    // The coarse rows come in row by row (one bulk copy each), from the 16-byte aligned coarse column at or below the one
    // under the tile's first column (an x-tile starts one vector left of its output columns, i.e. at an odd coarse column in
    // fp64): CPAD more elements per row than the TC/2 + 1 the tile needs at most
    // (x-tiled variant, XT; full-row tiles -- one contiguous chunk of CROWS rows per coarse plane -- keep the plain pitch TC/2)
    static constexpr int CPAD = 16 / (int)sizeof(T);
    static constexpr int CROWS = ZWY * ZR / 2 + 2;
    template <bool XT> static constexpr int csx_v = XT ? TC / 2 + CPAD : TC / 2;             // coarse row pitch in shared memory
    template <bool XT> static constexpr int cinp_v = XT ? CROWS * (TC / 2 + CPAD) : CROWS * (TC / 2) + CPAD;   // (+ the element after the last row)
};
constexpr int ZQB = 200;   // capacity of the work partition table: at most ZQB-1 CTAs
constexpr int ZNIN = 4;   // input ring depth (planes); 3 in the prolongation-fused variant (shared memory pays for the coarse ring)
constexpr int ZNCE = 3;   // coarse-correction ring depth (planes), prolongation-fused variant only

template <int NIN> __device__ __forceinline__ int ring_slot(int pos) { return NIN == 4 ? (pos & 3) : pos % NIN; }
template <int NIN> __device__ __forceinline__ uint32_t ring_par(int pos) { return NIN == 4 ? (uint32_t)((pos >> 2) & 1) : (uint32_t)((pos / NIN) & 1); }

template <typename T>
struct __align__(16) ZVec {
    T v[ZV<T>::N];
};

template <typename T>
struct Patch {
    ZVec<T> r[ZV<T>::R];
};

template <typename T>
struct ZP {
    int sx, sy, nz;
    long long sp;
    const T* tab;       // 10*nz: cx|cy|diag|w | A|Bx|By|Bz|iw|wz   (mhs_api.cu build_hierarchy)
    T cz, a2, rho;      // 1/hz^2, alpha^2, Bx/By = hy^2/hx^2
    int WX, WY;         // warps per tile along x / y
    int TC, COUT, ntx;  // tile columns, output columns per tile, tiles along x (1: the tile is a full row)
    int STEP, nty;      // distance between tiles along y (rows), tiles along y
    int NP;             // interior planes nz-2
    long long items;    // ntx*nty*NP
    int zcap;           // planes of the shared coefficient table
    const T* ec;        // prolongation-fused variant: the coarse-grid correction (aliased layout, pitch sx/2), else null
    long long csp;      //   its plane stride
    int in_plane;       // elements of one ring slot: (WY*ZR + 2) rows x TC (also the size of an exchange plane)
    int coef_bytes;     // bytes reserved for the coefficient table (multiple of 128)
    int qb[ZQB];        // CTA b works on the items [qb[b], qb[b+1]) of the linearised (tile, plane) list (zpartition)
    int useg, nunits;   // useg > 0: "unit" mode instead -- every tile is cut into the same useg z-segments, unit u = (segment
                        // u / ntiles, tile u % ntiles), CTA b takes the units b, b + gridDim.x, ...: y-neighbouring tiles are walked
                        // through the same planes at the same time (zcfg_make, "aligned segments")
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
// MHS_L2_HINT = 1: the iterate a smoothing pass reads is dead once read (the pass writes the other ping-pong buffer and the
// next pass reads THAT one), so its lines are marked evict-first in the L2: what stays in the 126 MB L2 at the end of a pass is
// mostly the iterate it has just written, which the next kernel (residual + restriction, or the next pass) reads back.
#ifndef MHS_L2_HINT
#define MHS_L2_HINT 0
#endif
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
#if MHS_L2_HINT
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
#else
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
#endif
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

template <typename T>
__device__ __forceinline__ ZVec<T> zld(const T* p) { return *reinterpret_cast<const ZVec<T>*>(p); }
template <typename T>
__device__ __forceinline__ void zst(T* p, const ZVec<T>& a) { *reinterpret_cast<ZVec<T>*>(p) = a; }
// MHS_ST_HINT: 1 = st.global.cs (streaming), 2 = L2::evict_first policy on the output stores of the fp64 passes
#ifndef MHS_ST_HINT
#define MHS_ST_HINT 0
#endif
__device__ __forceinline__ void zst_out(double* p, const ZVec<double>& a)
{
#if MHS_ST_HINT == 1
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(a.v[0]), "d"(a.v[1]) : "memory");
#elif MHS_ST_HINT == 2
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(a.v[0]), "d"(a.v[1]), "l"(pol) : "memory");
#else
    *reinterpret_cast<ZVec<double>*>(p) = a;
#endif
}

// Per-plane coefficients of one sweep (warp-uniform, read from the shared table).
//   fp64 (expanded update):  u' = A u + By (rho (e+w) + (n+s)) + Bz (up+dn) + wz f ;  iw2 = (D/omega)^2 for the norm
//   fp32 (difference form):  u' = u + wz (f - L u) with cx, cy per plane
template <typename T> struct ZCoef;
template <> struct ZCoef<double> {
    double A, By, Bz, wz, iw2;
    __device__ __forceinline__ void load(const double* ck, bool rhs, bool norm)
    {
        const double2 a = *reinterpret_cast<const double2*>(ck);
        const double2 b = *reinterpret_cast<const double2*>(ck + 2);
        A = a.x; By = a.y; Bz = b.x; wz = rhs ? b.y : 0.0;
        iw2 = norm ? ck[4] : 0.0;
    }
};
template <> struct ZCoef<float> {
    float cx, cy, wz;
    __device__ __forceinline__ void load(const float* ck, bool, bool)
    {
        const float4 a = *reinterpret_cast<const float4*>(ck);
        cx = a.x; cy = a.y; wz = a.z;
    }
};

__device__ __forceinline__ double zc_iw2(const ZCoef<double>& k) { return k.iw2; }
__device__ __forceinline__ double zc_iw2(const ZCoef<float>&) { return 0.0; }

// One Jacobi update of one row of a thread's patch.  c: the row's centre values, w/e: the elements left / right of
// the vector, n/s: the rows above / below, up/dn: the planes above / below, f: right-hand side.  rs (fp32 only): the
// sum of the squared residuals of the row, without element 0 when it is a wall (cw0).
// ISO: hx == hy, i.e. rho == 1: fma(1, a, b) is a + b rounded once, so the plain sum gives the same bits with one fp64
// instruction less per update (6 instead of 7) -- the fp64 pipe is the kernel's second busiest unit.
template <bool HAS_RHS, bool ISO>
__device__ __forceinline__ void jac_row(const ZCoef<double>& k, double rho, double, double, const ZVec<double>& c, double w, double e,
                                        const ZVec<double>& n, const ZVec<double>& s, const ZVec<double>& up, const ZVec<double>& dn,
                                        const ZVec<double>& f, ZVec<double>& o, bool, float&)
{
    double o0 = k.A * c.v[0], o1 = k.A * c.v[1];
    const double h0 = ISO ? (c.v[1] + w) + (n.v[0] + s.v[0]) : fma(rho, c.v[1] + w, n.v[0] + s.v[0]);
    const double h1 = ISO ? (e + c.v[0]) + (n.v[1] + s.v[1]) : fma(rho, e + c.v[0], n.v[1] + s.v[1]);
    o0 = fma(k.By, h0, o0);
    o1 = fma(k.By, h1, o1);
    o0 = fma(k.Bz, up.v[0] + dn.v[0], o0);
    o1 = fma(k.Bz, up.v[1] + dn.v[1], o1);
    if (HAS_RHS) {
        o0 = fma(k.wz, f.v[0], o0);
        o1 = fma(k.wz, f.v[1], o1);
    }
    o.v[0] = o0;
    o.v[1] = o1;
}

template <bool HAS_RHS, bool ISO>
__device__ __forceinline__ void jac_row(const ZCoef<float>& k, float, float cz, float a2, const ZVec<float>& c, float w, float e,
                                        const ZVec<float>& n, const ZVec<float>& s, const ZVec<float>& up, const ZVec<float>& dn,
                                        const ZVec<float>& f, ZVec<float>& o, bool cw0, float& rs)
{
    float ra = 0.f;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float cc = c.v[q];
        const float ww = q == 0 ? w : c.v[q - 1 < 0 ? 0 : q - 1];
        const float ee = q == 3 ? e : c.v[q + 1 > 3 ? 3 : q + 1];
        float lu = k.cx * lap1<float>(ee, ww, cc) + k.cy * lap1<float>(n.v[q], s.v[q], cc);
        lu += cz * lap1<float>(up.v[q], dn.v[q], cc) + a2 * cc;
        const float res = (HAS_RHS ? f.v[q] : 0.f) - lu;
        if (q > 0 || !cw0) ra = fmaf(res, res, ra);   // a wall element has no residual
        o.v[q] = cc + k.wz * res;
    }
    rs = ra;
}

// ------------------------------------------------------------------------------------------------
// S sweeps.  ZERO: the input iterate is identically zero (coarse-grid correction, first pre-sweep):
// sweep 1 is u = (omega/D) rhs and no input plane is read at all.
// ------------------------------------------------------------------------------------------------
// shared-memory access by 32-bit shared-space address (keeps addresses in one register each)
template <typename T> __device__ __forceinline__ ZVec<T> lds_vec(uint32_t a);
template <> __device__ __forceinline__ ZVec<double> lds_vec<double>(uint32_t a)
{
    ZVec<double> v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.v[0]), "=d"(v.v[1]) : "r"(a));
    return v;
}
template <> __device__ __forceinline__ ZVec<float> lds_vec<float>(uint32_t a)
{
    ZVec<float> v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.v[0]), "=f"(v.v[1]), "=f"(v.v[2]), "=f"(v.v[3]) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_vec(uint32_t a, const ZVec<double>& v)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.v[0]), "d"(v.v[1]) : "memory");
}
__device__ __forceinline__ void sts_vec(uint32_t a, const ZVec<float>& v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.v[0]), "f"(v.v[1]), "f"(v.v[2]), "f"(v.v[3]) : "memory");
}
template <typename T> __device__ __forceinline__ T lds_one(uint32_t a);
template <> __device__ __forceinline__ double lds_one<double>(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
template <> __device__ __forceinline__ float lds_one<float>(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void mbar_wait32(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "ZW2_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra ZW2_DONE;\n"
        "bra ZW2_WAIT;\n"
        "ZW2_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

template <typename T>
struct ZCtx {
    const T* f1;                  // global, per thread: (patch row 0, element 0) of the rhs plane sweep 1 reads in this step
    T* o_last;                    // global, per thread: same node of the plane the last sweep writes in this step
    uint32_t bars;                // shared-space addresses: mbarriers,
    uint32_t coef;                //   coefficient record of the plane sweep 1 makes in this step,
    uint32_t in_own;              //   ring slot 0 + offset of the patch,
    uint32_t ex_own;              //   exchange plane 0 + offset of the patch
    int t;                        // the step: input plane t arrives, sweep 1 makes plane t-1, sweep 2 plane t-2
    int kb, nout;                 // output planes [kb, kb+nout)
    int kend_in;                  // last input plane of the segment
    int zoff;                     // ring position of input plane k is zoff + k
    int omask;                    // rows of the patch that are stored (output rows, output columns)
    bool cw0;                     // element 0 of the patch is a wall column
    bool swp;                     // this lane fetches its x-neighbours in swapped order (see z_step)
    uint32_t eo1, eo2;            // byte offsets, from a row's vector, of the first / second x-neighbour load
    double acc;
    // prolongation-fused variant
    uint32_t in_base, ce_base;    // shared-space addresses of ring slot 0 / coarse ring slot 0
    uint32_t ce_own;              // byte offset, inside a coarse slot, of (coarse row jrow0>>1, coarse column of element 0)
    int czoff, cnext;             // ring position of coarse plane K is czoff + K; next coarse plane to request
    int jt, Jb;                   // first patch row of the tile (always odd); first coarse row held in a coarse slot
    int cbase;                    // first coarse column held in a coarse slot
    uint32_t c0a, c1a;            // this step's two coarse planes (shared-space addresses), set by z_prolong
    // ring positions kept incrementally (a ring of 3 would otherwise cost a division per use and step):
    int rs;                       // ring slot of plane t (== (zoff + t) % NIN), rp: its mbarrier parity
    uint32_t rp;
    int cs0;                      // prolongation-fused variant: coarse slot of coarse plane t >> 1, cp0: its parity
    uint32_t cp0;
    // the halo vector this thread corrects (prolongation-fused variant), fixed per segment
    bool h_ok;                    //   it exists and lies on an interior row
    uint32_t h_a, h_co, h_dj;     //   byte offsets: inside a ring slot, inside a coarse slot, to the second coarse row
    bool h_c0;                    //   its element 0 is a wall column
    bool corr;                    // the plane that arrives in this step takes a correction (interior plane)
    bool wrow;                    // the last patch row of this thread is the wall row j = sy (last tile along y): held at zero
};

// warp 0: request input plane `k` of the tile into ring slot nload % NIN
template <typename T, int WXT, int NIN>
__device__ __forceinline__ void z_issue(const ZP<T>& p, const T* tile_src, uint32_t bars, T* IN, int slot, int k)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    constexpr int TCc = ZG<T, WXT>::TC, INP = ZG<T, WXT>::INP;
    T* dst = IN + (size_t)slot * INP;
    const T* src = tile_src + p.sp * k;
    const uint32_t plane_bytes = (uint32_t)INP * sizeof(T);
    uint64_t* bar = reinterpret_cast<uint64_t*>(__cvta_shared_to_generic(bars)) + slot;
    const int lane = threadIdx.x & 31;
    if (p.ntx == 1) {
        if (lane == 0) {
            mbar_expect_tx(bar, plane_bytes);
            bulk_g2s(dst, src, plane_bytes, bar);
        }
    } else {
        if (lane == 0) mbar_expect_tx(bar, plane_bytes);
        __syncwarp();
        const int rows_in = ZWY * ZR + 2;
        for (int r = lane; r < rows_in; r += 32)
            bulk_g2s(dst + r * TCc, src + (long long)r * p.sx, (uint32_t)(TCc * sizeof(T)), bar);
    }
}

// Prolongation-fused variant, warp 0: make sure every coarse plane up to the one fine plane `kfine` needs has been requested.
// Coarse plane K (rows Jb .. Jb+CROWS-1, contiguous: full-row tiles) goes to coarse slot (czoff + K) % ZNCE; its mbarrier
// follows the NIN barriers of the input ring.
template <typename T, int WXT, int NIN, int PRO>
__device__ __forceinline__ void c_request(const ZP<T>& p, ZCtx<T>& z, int kfine)
{
    constexpr int CINP = ZG<T, WXT>::template cinp_v<PRO == 2>, CSX = ZG<T, WXT>::template csx_v<PRO == 2>;
    if (threadIdx.x >= 32) return;      // (cnext lives in warp 0)
    const int klast = min(min(kfine, z.kend_in), p.nz - 2);
    if (klast < 1) return;
    const int kneed = (klast + 1) >> 1;
    while (z.cnext <= kneed) {
        {
            const int cpos = z.czoff + z.cnext;
            const int slot = cpos % ZNCE;
            uint64_t* bar = reinterpret_cast<uint64_t*>(__cvta_shared_to_generic(z.bars)) + NIN + slot;
            T* dst = reinterpret_cast<T*>(__cvta_shared_to_generic(z.ce_base)) + (size_t)slot * CINP;
            const T* src = p.ec + p.csp * z.cnext + (long long)(p.sx >> 1) * z.Jb + (PRO == 2 ? z.cbase : 0);
            const int lane = (int)threadIdx.x;
            if (PRO == 2) {      // x-tiles: the coarse rows under the tile are not contiguous -- one copy per row
                if (lane == 0) mbar_expect_tx(bar, (uint32_t)(CINP * sizeof(T)));
                __syncwarp();
                if (lane < ZG<T, WXT>::CROWS) bulk_g2s(dst + lane * CSX, src + (long long)lane * (p.sx >> 1), (uint32_t)(CSX * sizeof(T)), bar);
            } else if (lane == 0) {
                mbar_expect_tx(bar, (uint32_t)(CINP * sizeof(T)));
                bulk_g2s(dst, src, (uint32_t)(CINP * sizeof(T)), bar);
            }
        }
        ++z.cnext;
    }
}

// Per-plane coefficients of one sweep (warp-uniform, read from the shared table).
//   fp64 (expanded update):  u' = A u + By (rho (e+w) + (n+s)) + Bz (up+dn) + wz f ;  iw2 = (D/omega)^2 for the norm
//   fp32 (difference form):  u' = u + wz (f - L u) with cx, cy per plane
__device__ __forceinline__ void zc_load(ZCoef<double>& k, uint32_t a, bool rhs, bool norm)
{
    const ZVec<double> x = lds_vec<double>(a);
    k.A = x.v[0]; k.By = x.v[1];
    if (rhs) {
        const ZVec<double> y = lds_vec<double>(a + 16);
        k.Bz = y.v[0]; k.wz = y.v[1];
    } else {
        k.Bz = lds_one<double>(a + 16); k.wz = 0.0;
    }
    k.iw2 = norm ? lds_one<double>(a + 32) : 0.0;
}
__device__ __forceinline__ void zc_load(ZCoef<float>& k, uint32_t a, bool, bool)
{
    const ZVec<float> x = lds_vec<float>(a);
    k.cx = x.v[0]; k.cy = x.v[1]; k.wz = x.v[2];
}

// End of a plane step: the ring slot of plane t-1 and the exchange plane of t-2 have been read by everybody.
template <typename T, int WXT, bool ZERO, int PRO>
__device__ __forceinline__ void z_advance(const ZP<T>& p, ZCtx<T>& z, const T* tile_src, T* IN, bool may_issue)
{
    constexpr int NIN = PRO ? 3 : ZNIN;
    __syncthreads();
    if (!ZERO && may_issue) {
        const int k = z.t + NIN - 1;      // the slot of plane t-1 is free: request plane t+NIN-1 into it
        if (k <= z.kend_in) {
            // (zoff + k) % NIN is the slot of plane t-1
            if (threadIdx.x < 32) z_issue<T, WXT, NIN>(p, tile_src, z.bars, IN, z.rs == 0 ? NIN - 1 : z.rs - 1, k);
            if (PRO) c_request<T, WXT, NIN, PRO>(p, z, k + 1);   // (one plane ahead: the coarse plane is there when its fine plane lands)
        }
    }
    ++z.t;
    if (++z.rs == NIN) { z.rs = 0; z.rp ^= 1u; }
    if (PRO && !(z.t & 1)) {            // t became even: t >> 1 moved on
        if (++z.cs0 == ZNCE) { z.cs0 = 0; z.cp0 ^= 1u; }
    }
}

// ------------------------------------------------------------------------------------------------
// Prolongation-fused variant, "stage 0": the trilinear correction u += P e_c (a6) is applied to input plane t IN PLACE in
// its ring slot as soon as it has arrived -- own patch rows by their owner, the two halo rows of the tile by one vector
// per thread -- so that the sweeps read corrected values everywhere and the separate prolongation pass (read u, write u)
// disappears.  Nobody but the owner reads plane t's slot before the barrier that ends the step.  Interior planes, rows and
// columns only (walls and the planes k = 0, nz-1 carry no correction).  Coarse operands come from the coarse ring.
//   u(i,j,k) += 1/8 * sum over the 2x2x2 coarse nodes ((i,i+1)>>1, (j,j+1)>>1, (k,k+1)>>1)
// ------------------------------------------------------------------------------------------------
template <typename T, int WXT, int JP, int PRO>
__device__ __forceinline__ void z_prolong_rows(const ZCtx<T>& z, uint32_t a_pl, uint32_t c0a, uint32_t c1a)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    constexpr int V = ZV<T>::N, VC = V / 2;
    constexpr uint32_t ES = sizeof(T);
    constexpr uint32_t rowb = (uint32_t)ZG<T, WXT>::TC * ES, crowb = (uint32_t)ZG<T, WXT>::template csx_v<PRO == 2> * ES;
    constexpr int NJ = (JP + ZR) / 2 + 1;          // coarse rows under the ZR patch rows
    T cz[NJ][VC + 1];                              // the two coarse planes summed
#pragma unroll
    for (int q = 0; q < NJ; ++q)
#pragma unroll
        for (int m = 0; m <= VC; ++m)
            cz[q][m] = lds_one<T>(c0a + z.ce_own + q * crowb + m * ES) + lds_one<T>(c1a + z.ce_own + q * crowb + m * ES);
#pragma unroll
    for (int r = 0; r < ZR; ++r) {
        const int q0 = (JP + r) >> 1, q1 = (JP + r + 1) >> 1;
        ZVec<T> a = lds_vec<T>(a_pl + r * rowb);
        T c[VC + 1];
#pragma unroll
        for (int m = 0; m <= VC; ++m) c[m] = cz[q0][m] + cz[q1][m];
#pragma unroll
        for (int e = 0; e < V; ++e) {
            const T sum = (e & 1) ? (c[e >> 1] + c[(e >> 1) + 1]) : T(2) * c[e >> 1];
            if (e > 0 || !z.cw0) a.v[e] += T(0.125) * sum;
        }
        sts_vec(a_pl + r * rowb, a);
    }
}

template <typename T, int WXT, int NIN, bool ROWS, int PRO>
__device__ __forceinline__ void z_prolong(const ZP<T>& p, ZCtx<T>& z, int t, int slot)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    constexpr int V = ZV<T>::N, VC = V / 2;
    constexpr uint32_t ES = sizeof(T);
    constexpr int TC = ZG<T, WXT>::TC, NR = ZWY * ZR;
    constexpr uint32_t planeb = (uint32_t)ZG<T, WXT>::INP * ES, cplaneb = (uint32_t)ZG<T, WXT>::template cinp_v<PRO == 2> * ES;
    constexpr uint32_t crowb = (uint32_t)ZG<T, WXT>::template csx_v<PRO == 2> * ES;
    z.corr = false;
    if (t < 1 || t > p.nz - 2) return;
    z.corr = true;
    // coarse planes t >> 1 (slot cs0) and (t + 1) >> 1 (the next slot when t is odd)
    const int s0 = z.cs0;
    int s1 = s0;
    uint32_t q1 = z.cp0;
    if (t & 1) {
        if (++s1 == ZNCE) { s1 = 0; q1 ^= 1u; }
    }
    mbar_wait32(z.bars + 8 * (NIN + s0), z.cp0);
    mbar_wait32(z.bars + 8 * (NIN + s1), q1);
    const uint32_t c0a = z.ce_base + (uint32_t)s0 * cplaneb, c1a = z.ce_base + (uint32_t)s1 * cplaneb;
    const uint32_t a_pl = z.in_own + (uint32_t)slot * planeb;
    z.c0a = c0a; z.c1a = c1a;
    if (ROWS) z_prolong_rows<T, WXT, 1, PRO>(z, a_pl, c0a, c1a);     // (jt is odd and patch rows start ZR-aligned from it)
    // the halo rows of the tile (fine rows jt-1 and jt+NR): one vector per thread (which one: fixed per segment, z.h_*)
    if (z.h_ok) {
        const uint32_t a = z.in_base + (uint32_t)slot * planeb + z.h_a;
        const uint32_t co = z.h_co, dj = z.h_dj;
        const bool hv_in = !z.h_c0;
        ZVec<T> v = lds_vec<T>(a);
        T c[VC + 1];
#pragma unroll
        for (int m = 0; m <= VC; ++m)
            c[m] = (lds_one<T>(c0a + co + m * ES) + lds_one<T>(c1a + co + m * ES)) +
                   (lds_one<T>(c0a + co + dj + m * ES) + lds_one<T>(c1a + co + dj + m * ES));
#pragma unroll
        for (int e = 0; e < V; ++e) {
            const T sum = (e & 1) ? (c[e >> 1] + c[(e >> 1) + 1]) : T(2) * c[e >> 1];
            if (e > 0 || hv_in) v.v[e] += T(0.125) * sum;
        }
        sts_vec(a, v);
    }
    (void)TC; (void)NR; (void)crowb; (void)VC;
}

// First step of a segment (t = kstart): nothing to compute yet, plane kstart becomes the centre plane.
template <typename T, int WXT, bool ZERO, int PRO>
__device__ __forceinline__ void z_first(const ZP<T>& p, ZCtx<T>& z, const T* tile_src, T* IN, Patch<T>& dn0)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    constexpr int NIN = PRO ? 3 : ZNIN;
    if (!ZERO) {
        mbar_wait32(z.bars + 8 * z.rs, z.rp);
        if (PRO) z_prolong<T, WXT, NIN, true, PRO>(p, z, z.t, z.rs);
        const uint32_t a = z.in_own + (uint32_t)z.rs * (uint32_t)(ZG<T, WXT>::INP * sizeof(T));
#pragma unroll
        for (int r = 0; r < ZR; ++r) dn0.r[r] = lds_vec<T>(a + r * (uint32_t)(ZG<T, WXT>::TC * sizeof(T)));
    }
    z_advance<T, WXT, ZERO, PRO>(p, z, tile_src, IN, false);
}

// pa += d0^2 + d1^2 where `on` is set: predicated FMAs (written as a select ptxas makes 2 FSEL per value of them)
__device__ __forceinline__ void norm_acc(double& pa, double& pb, double d0, double d1, int on)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %4, 0;\n\t@p fma.rn.f64 %0, %2, %2, %0;\n\t@p fma.rn.f64 %1, %3, %3, %1;\n\t}"
        : "+d"(pa), "+d"(pb)
        : "d"(d0), "d"(d1), "r"(on));
}

// The rows of one plane step in fp64 (not the zero-guess variant).  The update is evaluated as
//     u' = [A c + By h + Bz dn (+ wz f)] + Bz up,        h = rho (e + w) + (n + s)
// i.e. everything but the last FMA is independent of the plane that arrives in this step (stage 1) and of the sweep-1
// value made in this step (stage 2).  Two things follow.  (i) The bracket of row r+1 is formed while row r is finished, so
// the shared-memory round trip of `up` and the stage 1 -> stage 2 dependency each cost one FMA of latency instead of an
// add + an FMA.  (ii) `dn` is dead once the bracket exists: the arriving plane is loaded straight into the registers of dn0
// and the sweep-1 result is produced straight into those of dn1, which is what they have to become for the next step --
// the 64 register moves per step that `dn0 = up; dn1 = o1` used to cost are gone.
// A wall column (element 0 of the first vector of a row) stays exactly zero through its coefficients: its own value and its
// z- and y-neighbours are walls (zero), so with By = wz = 0 for that element the update returns 0 -- no select per row.
template <int WXT, int S, bool HAS_RHS, bool NORM, int PRO, bool ISO>
__device__ __forceinline__ void z_rows64(const ZP<double>& p, ZCtx<double>& z, const ZCoef<double>& k1, const ZCoef<double>& k2, Patch<double>& dn0,
                                         const Patch<double>& c0, Patch<double>& dn1, const Patch<double>& c1, uint32_t a_new, uint32_t a_cen,
                                         uint32_t a_exw, uint32_t a_exr, int m1, int m2, double& pa)
{
    using T = double;
    constexpr int ZR = ZV<T>::R;
    constexpr uint32_t rowb = (uint32_t)ZG<T, WXT>::TC * 8u;
    const double By1a = z.cw0 ? 0.0 : k1.By, wz1a = z.cw0 ? 0.0 : k1.wz;
    const double By2a = z.cw0 ? 0.0 : k2.By, wz2a = z.cw0 ? 0.0 : k2.wz;
    const uint32_t a_cen1 = a_cen + z.eo1, a_cen2 = a_cen + z.eo2, a_exr1 = a_exr + z.eo1, a_exr2 = a_exr + z.eo2;
    struct Nb {
        T q1, q2, q3, q4;        // x-neighbours as loaded: (w, e) or, on the lanes with z.swp, (e, w); stage 1 | stage 2
        ZVec<T> f1, f2;
    };
    auto load_nb = [&](int r, Nb& q) {
        const long long grow = (long long)r * p.sx;
        q.q1 = lds_one<T>(a_cen1 + r * rowb);
        q.q2 = lds_one<T>(a_cen2 + r * rowb);
        if (HAS_RHS) q.f1 = zld(z.f1 + grow);
        if (S == 2) {
            q.q3 = lds_one<T>(a_exr1 + r * rowb);
            q.q4 = lds_one<T>(a_exr2 + r * rowb);
            if (HAS_RHS) q.f2 = zld(z.f1 - p.sp + grow);
        }
    };
    // the bracket of one row of one stage
    auto bracket = [&](const ZCoef<T>& k, double Bya, double wza, const ZVec<T>& c, T w, T e, const ZVec<T>& n, const ZVec<T>& s2,
                       const ZVec<T>& dn, const ZVec<T>& f) {
        ZVec<T> a;
        const double h0 = ISO ? (c.v[1] + w) + (n.v[0] + s2.v[0]) : fma(p.rho, c.v[1] + w, n.v[0] + s2.v[0]);
        const double h1 = ISO ? (e + c.v[0]) + (n.v[1] + s2.v[1]) : fma(p.rho, e + c.v[0], n.v[1] + s2.v[1]);
        a.v[0] = fma(k.Bz, dn.v[0], k.A * c.v[0]);
        a.v[1] = fma(k.Bz, dn.v[1], k.A * c.v[1]);
        a.v[0] = fma(Bya, h0, a.v[0]);
        a.v[1] = fma(k.By, h1, a.v[1]);
        if (HAS_RHS) {
            a.v[0] = fma(wza, f.v[0], a.v[0]);
            a.v[1] = fma(k.wz, f.v[1], a.v[1]);
        }
        return a;
    };
    const ZVec<T> lo1 = lds_vec<T>(a_cen - rowb), hi1 = lds_vec<T>(a_cen + ZR * rowb);     // rows -1 and ZR of the centre planes
    ZVec<T> lo2, hi2;
    if (S == 2) { lo2 = lds_vec<T>(a_exr - rowb); hi2 = lds_vec<T>(a_exr + ZR * rowb); }
    Nb nb[2];
    ZVec<T> acc1[2], acc2[2];
    // prolongation-fused variant: the two coarse planes of this step summed, per coarse row under the patch (loaded as needed);
    // planes without a correction (k = 0, nz-1, the idle step) run the same code with the weights 0 on whatever finite
    // numbers the coarse ring holds (it is zero-filled at the start of the kernel)
    constexpr uint32_t crowb = (uint32_t)ZG<T, WXT>::template csx_v<PRO == 2> * 8u;
    T cz[ZR / 2 + 1][2], czr[ZR / 2 + 1][4];
    const T cs1 = (PRO && z.corr) ? 0.125 : 0.0, cs2 = (PRO && z.corr) ? 0.25 : 0.0;
    const uint32_t cb0 = z.c0a + z.ce_own, cb1 = z.c1a + z.ce_own;
    auto czload = [&](int q) {    // (issued well ahead of czsum: a store to shared memory sits between every two rows, and no
                                  //  load can be moved up across it by the assembler)
        czr[q][0] = lds_one<T>(cb0 + q * crowb); czr[q][1] = lds_one<T>(cb1 + q * crowb);
        czr[q][2] = lds_one<T>(cb0 + q * crowb + 8); czr[q][3] = lds_one<T>(cb1 + q * crowb + 8);
    };
    auto czsum = [&](int q) { cz[q][0] = czr[q][0] + czr[q][1]; cz[q][1] = czr[q][2] + czr[q][3]; };
    auto pre = [&](int r) {     // brackets of row r; afterwards dn0.r[r] and dn1.r[r] are dead and take their new contents
        const Nb& q = nb[r & 1];
        const T w1 = z.swp ? q.q2 : q.q1, e1 = z.swp ? q.q1 : q.q2;
        acc1[r & 1] = bracket(k1, By1a, wz1a, c0.r[r], w1, e1, r == ZR - 1 ? hi1 : c0.r[r + 1 < ZR ? r + 1 : r], r == 0 ? lo1 : c0.r[r > 0 ? r - 1 : 0],
                              dn0.r[r], q.f1);
        if (!PRO) dn0.r[r] = lds_vec<T>(a_new + r * rowb);      // plane t: `up` now, the centre plane of the next step
        if (PRO) {
            // prolongation folded in (a6): plane t takes u += P e_c as it is read, and goes back corrected to its ring slot,
            // where the neighbours read it in the next step.  jt is odd: patch row r lies between the coarse rows (r+1)>>1
            // and (r+2)>>1 of the tile's coarse rows (coincident when they are equal).  A wall column needs no test: the
            // coarse wall value it would take is zero.
            const int q0 = (1 + r) >> 1, q1 = (2 + r) >> 1;
            if (r == 0) { czsum(0); czsum(1); }
            else if (q1 != q0) czsum(q1);
            const T e0 = cz[q0][0] + cz[q1][0], e1 = cz[q0][1] + cz[q1][1];
            // (the plane's row loaded two rows ahead of this point into a buffer of its own bought nothing -- 82.8 -> 82.4 us --
            //  and cost eight registers: 64 bytes of spills in the x-tiled variant)
            const ZVec<T> raw = lds_vec<T>(a_new + r * rowb);
            dn0.r[r].v[0] = fma(cs2, e0, raw.v[0]);
            dn0.r[r].v[1] = fma(cs1, e0 + e1, raw.v[1]);
            sts_vec(a_new + r * rowb, dn0.r[r]);
            if (r + 2 < ZR && ((4 + r) >> 1) != ((3 + r) >> 1)) czload((4 + r) >> 1);      // the coarse row that row r+2 adds
        }
        if (S == 2) {
            const T w2 = z.swp ? q.q4 : q.q3, e2 = z.swp ? q.q3 : q.q4;
            acc2[r & 1] = bracket(k2, By2a, wz2a, c1.r[r], w2, e2, r == ZR - 1 ? hi2 : c1.r[r + 1 < ZR ? r + 1 : r],
                                  r == 0 ? lo2 : c1.r[r > 0 ? r - 1 : 0], dn1.r[r], q.f2);
        }
    };
    double pn[4] = {0.0, 0.0, 0.0, 0.0};     // four partial sums of the norm: dependency chains of 4 FMAs instead of 16
    if (PRO) {
        czload(0); czload(1);                  // (row r+2's new coarse row is requested while row r is corrected)
    }
    load_nb(0, nb[0]);
    if (ZR > 1) load_nb(1, nb[1]);
    pre(0);
#pragma unroll
    for (int r = 0; r < ZR; ++r) {
        const long long grow = (long long)r * p.sx;
        if (r + 2 < ZR) load_nb(r + 2, nb[r & 1]);     // (ahead of pre(): its store of the corrected row would pin these loads behind it)
        if (r + 1 < ZR) pre(r + 1);
        // ---------------- stage 1: sweep-1 values of row r of plane t-1 ----------------
        ZVec<T> o1;
        o1.v[0] = fma(k1.Bz, dn0.r[r].v[0], acc1[r & 1].v[0]);
        o1.v[1] = fma(k1.Bz, dn0.r[r].v[1], acc1[r & 1].v[1]);
        if (r == ZR - 1 && z.wrow) o1.v[0] = o1.v[1] = 0.0;    // the wall row j = sy, when the tile holds it as a patch row
        if (NORM) norm_acc(pn[(2 * r) & 3], pn[(2 * r + 1) & 3], o1.v[0] - c0.r[r].v[0], o1.v[1] - c0.r[r].v[1], m1 & (1 << r));
        if (S == 1) {
            if (m1 & (1 << r)) zst_out(z.o_last + grow, o1);
        } else {
            sts_vec(a_exw + r * rowb, o1);
            // ---------------- stage 2: sweep-2 values of row r of plane t-2 ----------------
            ZVec<T> o2;
            o2.v[0] = fma(k2.Bz, o1.v[0], acc2[r & 1].v[0]);
            o2.v[1] = fma(k2.Bz, o1.v[1], acc2[r & 1].v[1]);
            if (m2 & (1 << r)) zst_out(z.o_last + grow, o2);
            dn1.r[r] = o1;  // becomes the sweep-1 centre plane of the next step
        }
    }
    if (NORM) pa = (pn[0] + pn[1]) + (pn[2] + pn[3]);
}

// One plane step, t > kstart.  Input planes of the patch: dn0 = t-2, c0 = t-1 (plane t is read from its ring
// slot); sweep-1 planes: dn1 = t-3, c1 = t-2.  On return dn0 holds plane t and dn1 holds sweep-1 plane t-1: the
// caller swaps the names (steps come in pairs).
template <typename T, int WXT, int S, bool HAS_RHS, bool ZERO, bool NORM, int PRO, bool ISO>
__device__ __forceinline__ void z_step(const ZP<T>& p, ZCtx<T>& z, const T* tile_src, T* IN, Patch<T>& dn0, const Patch<T>& c0, Patch<T>& dn1,
                                       const Patch<T>& c1)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    constexpr int V = ZV<T>::N;
    constexpr uint32_t ES = sizeof(T);
    constexpr uint32_t rowb = (uint32_t)ZG<T, WXT>::TC * ES;
    constexpr uint32_t planeb = (uint32_t)ZG<T, WXT>::INP * ES;
    const int t = z.t;
    const bool in1 = (unsigned)(t - 1 - z.kb) < (unsigned)z.nout;   // plane t-1 is an output plane of this segment
    const bool in2 = (unsigned)(t - 2 - z.kb) < (unsigned)z.nout;
    const bool fresh = !ZERO && t <= z.kend_in;                      // a new input plane arrives in this step
    // !fresh (only the step after the top plane): the slot holds an older plane -- finite numbers that meet Bz = 0
    constexpr int NIN = PRO ? 3 : ZNIN;
    const uint32_t a_new = z.in_own + (uint32_t)z.rs * planeb;                                   // plane t
    const uint32_t a_cen = z.in_own + (uint32_t)(z.rs == 0 ? NIN - 1 : z.rs - 1) * planeb;       // plane t-1
    const uint32_t a_exw = z.ex_own + (uint32_t)(t & 1) * planeb;                      // sweep-1 plane t-1 (written now)
    const uint32_t a_exr = z.ex_own + (uint32_t)((t & 1) ^ 1) * planeb;                // sweep-1 plane t-2 (written a step ago)
    if (fresh) mbar_wait32(z.bars + 8 * z.rs, z.rp);
    if (PRO) z.corr = false;
    if (PRO && fresh) z_prolong<T, WXT, NIN, sizeof(T) == 4, PRO>(p, z, t, z.rs);   // fp64: own rows inside the row loop
    ZCoef<T> k1, k2;
    zc_load(k1, z.coef, HAS_RHS, NORM);
    if (S == 2) zc_load(k2, z.coef - ZV<T>::NCO * ES, HAS_RHS, false);
    const int m1 = in1 ? z.omask : 0, m2 = in2 ? z.omask : 0;
    double pa = 0.0;
    float pf = 0.f;
    // Everything a row needs from memory, fetched ONE ROW AHEAD of the arithmetic (the loop is fully unrolled, so the
    // two sets are just names): the loads of row r+1 are in flight while row r is computed, instead of each row
    // exposing a shared-memory round trip at its first use.
    struct RowIn {
        ZVec<T> up0, edge1, edge2, f1, f2;
        T w, e, w2, e2;
    };
    // x-neighbours (the element left of the vector, w, and the one right of it, e) are single elements 16 bytes apart
    // from lane to lane: a warp-wide load of all the w (or all the e) touches only every other 8-byte bank pair (fp64; one
    // bank in four in fp32) and takes twice the wavefronts it needs -- measured, these loads were 40 % of the kernel's
    // shared-memory wavefronts, and the shared-memory pipe is its busiest unit.  So lanes 8-15 and 24-31 fetch e where the
    // others fetch w and the other way round in the second load: every half-warp then covers all banks.  The two values are
    // put back in order with selects (z.swp).
    const uint32_t a_cen1 = a_cen + z.eo1, a_cen2 = a_cen + z.eo2, a_exr1 = a_exr + z.eo1, a_exr2 = a_exr + z.eo2;
    auto load_row = [&](int r, RowIn& q) {
        const long long grow = (long long)r * p.sx;
        if (!ZERO) {
            q.up0 = lds_vec<T>(a_new + r * rowb);
            q.w = lds_one<T>(a_cen1 + r * rowb);
            q.e = lds_one<T>(a_cen2 + r * rowb);
            if (r == ZR - 1) q.edge1 = lds_vec<T>(a_cen + ZR * rowb);
            if (r == 0) q.edge1 = lds_vec<T>(a_cen - rowb);
        }
        if (HAS_RHS) q.f1 = zld(z.f1 + grow);
        if (S == 2) {
            q.w2 = lds_one<T>(a_exr1 + r * rowb);
            q.e2 = lds_one<T>(a_exr2 + r * rowb);
            if (r == ZR - 1) q.edge2 = lds_vec<T>(a_exr + ZR * rowb);
            if (r == 0) q.edge2 = lds_vec<T>(a_exr - rowb);
            if (HAS_RHS) q.f2 = zld(z.f1 - p.sp + grow);
        }
    };
    if constexpr (sizeof(T) == 8 && !ZERO) {
        z_rows64<WXT, S, HAS_RHS, NORM, PRO, ISO>(p, z, k1, k2, dn0, c0, dn1, c1, a_new, a_cen, a_exw, a_exr, m1, m2, pa);
    } else {
    RowIn rin[2];
    load_row(0, rin[0]);
#pragma unroll
    for (int r = 0; r < ZR; ++r) {
        const long long grow = (long long)r * p.sx;
        RowIn& in = rin[r & 1];
        if (r + 1 < ZR) load_row(r + 1, rin[(r + 1) & 1]);
        // ---------------- stage 1: sweep-1 values of row r of plane t-1 ----------------
        ZVec<T> o1;
        if (ZERO) {
#pragma unroll
            for (int e = 0; e < V; ++e) o1.v[e] = (r == ZR - 1 && z.wrow) ? T(0) : k1.wz * in.f1.v[e];
            if (z.cw0) o1.v[0] = T(0);
        } else {
            const ZVec<T> nn = r == ZR - 1 ? in.edge1 : c0.r[r + 1 < ZR ? r + 1 : r];
            const ZVec<T> ss = r == 0 ? in.edge1 : c0.r[r > 0 ? r - 1 : 0];
            float rs = 0.f;
            const T w1 = z.swp ? in.e : in.w, e1 = z.swp ? in.w : in.e;
            jac_row<HAS_RHS, ISO>(k1, p.rho, p.cz, p.a2, c0.r[r], w1, e1, nn, ss, in.up0, dn0.r[r], in.f1, o1, z.cw0, rs);
            if (z.cw0) o1.v[0] = c0.r[r].v[0];
            if (r == ZR - 1 && z.wrow) {
#pragma unroll
                for (int e = 0; e < V; ++e) o1.v[e] = T(0);
            }
            if (NORM && (m1 & (1 << r))) {
                if (sizeof(T) == 8) {
#pragma unroll
                    for (int q = 0; q < V; ++q) {
                        const double d = (double)o1.v[q] - (double)c0.r[r].v[q];
                        pa = fma(d, d, pa);
                    }
                } else {
                    pf += rs;
                }
            }
            dn0.r[r] = in.up0;     // becomes the centre plane of the next step
        }
        if (S == 1) {
            if (m1 & (1 << r)) zst(z.o_last + grow, o1);
        } else {
            sts_vec(a_exw + r * rowb, o1);
            // ---------------- stage 2: sweep-2 values of row r of plane t-2 ----------------
            ZVec<T> o2;
            const ZVec<T> nn = r == ZR - 1 ? in.edge2 : c1.r[r + 1 < ZR ? r + 1 : r];
            const ZVec<T> ss = r == 0 ? in.edge2 : c1.r[r > 0 ? r - 1 : 0];
            float rs;
            const T w2 = z.swp ? in.e2 : in.w2, e2 = z.swp ? in.w2 : in.e2;
            jac_row<HAS_RHS, ISO>(k2, p.rho, p.cz, p.a2, c1.r[r], w2, e2, nn, ss, o1, dn1.r[r], in.f2, o2, false, rs);
            if (z.cw0) o2.v[0] = c1.r[r].v[0];
            if (m2 & (1 << r)) zst(z.o_last + grow, o2);
            dn1.r[r] = o1;  // becomes the sweep-1 centre plane of the next step
        }
    }
    }
    if (NORM) {
        if (sizeof(T) == 8) z.acc = fma(zc_iw2(k1), pa, z.acc);   // pa == 0 unless plane t-1 is an output plane
        else z.acc += (double)pf;
    }
    z.coef += ZV<T>::NCO * ES;
    z.o_last += p.sp;
    if (HAS_RHS) z.f1 += p.sp;
    z_advance<T, WXT, ZERO, PRO>(p, z, tile_src, IN, true);
}

template <typename T, int WXT, int S, bool HAS_RHS, bool ZERO, bool NORM, int PRO, bool ISO>
__global__ void __launch_bounds__(WXT * ZV<T>::WY * 32, 1) k_zsweep(const __grid_constant__ ZP<T> p, const T* __restrict__ u, const T* __restrict__ rhs,
                                                    T* __restrict__ out, double* __restrict__ partial, const int* __restrict__ done)
{
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY; (void)ZR; (void)ZWY;
    static_assert(S == 1 || S == 2, "S sweeps per pass: 1 or 2");
    static_assert(!ZERO || HAS_RHS, "a zero iterate with a zero right-hand side stays zero");
    static_assert(!PRO || (!ZERO && !NORM), "the prolongation-fused pass is a post-smoothing pass");
    constexpr int NIN = PRO ? 3 : ZNIN;
    pdl_enter();
    if (done && *done) return;
    constexpr int V = ZV<T>::N;
    constexpr int NCO = ZV<T>::NCO;
    constexpr int H = S - 1;                               // rows a tile loses on each side to the later sweeps
    extern __shared__ __align__(128) unsigned char zsm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wx = warp % WXT, wy = warp / WXT;
    constexpr int TC = ZG<T, WXT>::TC, INP = ZG<T, WXT>::INP;
    constexpr int NR = ZWY * ZR;                           // patch rows of a tile
    // shared memory: [mbarriers: 128 B] [coefficients: a pad record + zcap records] [IN ring: NIN planes] [EX: 2 planes]
    // [PRO: coarse ring, ZNCE planes]
    uint64_t* bars = reinterpret_cast<uint64_t*>(zsm);
    T* coef = reinterpret_cast<T*>(zsm + 128) + NCO;       // record of plane kstart; the record before it is a pad
    T* IN = reinterpret_cast<T*>(zsm + 128 + p.coef_bytes);
    T* EX = IN + (size_t)(ZERO ? 0 : NIN) * INP;
    T* CE = EX + (size_t)2 * INP;

    if (!ZERO && threadIdx.x == 0) {
        for (int q = 0; q < NIN + (PRO ? ZNCE : 0); ++q) mbar_init(bars + q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (S == 2) {   // guard rows and never-written parts of the exchange planes must hold zeros (a wall row may sit there)
        for (int q = threadIdx.x; q < 2 * INP; q += blockDim.x) EX[q] = T(0);
    }
    if (threadIdx.x < NCO) coef[-NCO + (int)threadIdx.x] = T(0);
    if (PRO) {   // (planes without a correction read the coarse ring with zero weights: finite numbers, please)
        for (int q = threadIdx.x; q < ZNCE * ZG<T, WXT>::template cinp_v<PRO == 2>; q += blockDim.x) CE[q] = T(0);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes before the bulk copies into the same memory
    }
    __syncthreads();

    const int cx0 = (wx * 32 + lane) * V;                   // first column of this thread's vector inside the tile
    ZCtx<T> z;
    z.bars = smem_u32(bars);
    z.in_own = smem_u32(IN + (wy * ZR + 1) * TC + cx0);
    z.ex_own = smem_u32(EX + (wy * ZR + 1) * TC + cx0);
    z.acc = 0.0;
    z.swp = (lane & 8) != 0;
    z.eo1 = z.swp ? (uint32_t)(V * sizeof(T)) : (uint32_t)(0u - (uint32_t)sizeof(T));
    z.eo2 = z.swp ? (uint32_t)(0u - (uint32_t)sizeof(T)) : (uint32_t)(V * sizeof(T));
    z.in_base = smem_u32(IN);
    z.ce_base = PRO ? smem_u32(CE) : 0u;
    z.ce_own = 0; z.czoff = 0; z.cnext = 0; z.jt = 0; z.Jb = 0; z.cbase = 0;
    z.c0a = z.c1a = z.ce_base; z.corr = false; z.wrow = false;
    z.rs = 0; z.rp = 0; z.cs0 = 0; z.cp0 = 0; z.h_ok = false; z.h_a = z.h_co = z.h_dj = 0; z.h_c0 = false;
    int ring = 0;                                           // planes requested so far by this CTA (ring position)
    int cring = 0;                                          // coarse planes requested so far (PRO)
    const long long q0 = p.qb[blockIdx.x], q1 = p.qb[blockIdx.x + 1];

    const int ntiles_all = p.ntx * p.nty;
    int unit = (int)blockIdx.x;
    for (long long q = q0;;) {
        int tile, kb, ke;                                              // output planes [kb, ke) of tile `tile`
        if (p.useg > 0) {
            if (unit >= p.nunits) break;
            const int seg = unit / ntiles_all;
            tile = unit - seg * ntiles_all;
            kb = 1 + (int)((long long)p.NP * seg / p.useg);
            ke = 1 + (int)((long long)p.NP * (seg + 1) / p.useg);
            unit += (int)gridDim.x;
        } else {
            if (q >= q1) break;
            tile = (int)(q / p.NP);
            kb = 1 + (int)(q - (long long)tile * p.NP);
            ke = (int)min((long long)p.NP + 1, kb + (q1 - q));
            q += ke - kb;
        }
        const int ty = tile / p.ntx, tx = tile - ty * p.ntx;
        const int ct = p.ntx == 1 ? 0 : tx * p.COUT - V;              // first column of the tile
        // Tiles along y: patch rows [jt, jt+NR) are interior rows; the wall rows j = 0 / j = sy are only ever
        // read -- from the input halo row in sweep 1, from the (zero) guard row of the exchange plane in sweep 2.
        // (always odd; the last tile is pulled back so that its last patch row is the wall row j = sy, which it holds at zero)
        const int jt = min(1 + ty * p.STEP, p.sy - NR + 1);            // first patch row
        const int jlo = ty == 0 ? 1 : 1 + ty * p.STEP + H;             // rows [jlo, jhi) are this tile's output
        const int jhi = ty == p.nty - 1 ? p.sy : 1 + ty * p.STEP + NR - H;
        const int kstart = max(kb - S, 0);
        const int kend_in = min(ke - 1 + S, p.nz - 1);
        const T* tile_src = u + (long long)(jt - 1) * p.sx + ct;      // (row jt-1, col ct) of plane 0

        // per-plane coefficient records of this segment
        __syncthreads();   // the previous segment is done with the table
        for (int i = threadIdx.x; i < (kend_in - kstart + 2) * NCO; i += blockDim.x) {   // + a zero record for the idle step
            const int k = kstart + i / NCO, c = i % NCO;
            const T* t = p.tab;
            T v = T(0);
            if (k > kend_in) {
            } else if (sizeof(T) == 8) {
                // A | By | Bz | wz | iw^2 | -
                if (c == 0) v = t[4 * p.nz + k];
                else if (c == 1) v = t[6 * p.nz + k];
                else if (c == 2) v = t[7 * p.nz + k];
                else if (c == 3) v = t[9 * p.nz + k];
                else if (c == 4) v = t[8 * p.nz + k] * t[8 * p.nz + k];
            } else {
                // cx | cy | wz | -
                if (c < 2) v = t[c * p.nz + k];
                else if (c == 2) v = t[9 * p.nz + k];
            }
            coef[i] = v;
        }
        z.zoff = ring - kstart;
        z.rs = ring_slot<NIN>(ring);
        z.rp = ring_par<NIN>(ring);
        if (!ZERO) {
            const int n = min(NIN, kend_in - kstart + 1);
            if (warp == 0)
                for (int i = 0; i < n; ++i) z_issue<T, WXT, NIN>(p, tile_src, z.bars, IN, ring_slot<NIN>(ring + i), kstart + i);
            ring += kend_in - kstart + 1;
            if (PRO) {
                // coarse planes (kfirst >> 1) .. ((klast + 1) >> 1) serve the corrected fine planes kfirst .. klast
                z.kend_in = kend_in;
                z.jt = jt;
                z.Jb = (jt - 1) >> 1;
                z.cbase = PRO == 2 ? (ct >> 1) & ~(ZG<T, WXT>::CPAD - 1) : 0;
                const int kfirst = max(kstart, 1), klast = min(kend_in, p.nz - 2);
                z.cnext = kfirst >> 1;
                z.czoff = cring - z.cnext;
                {   // ring position of coarse plane kstart >> 1 (== kfirst >> 1)
                    const int p0 = z.czoff + (kstart >> 1);
                    z.cs0 = p0 % ZNCE;
                    z.cp0 = (uint32_t)((p0 / ZNCE) & 1);
                }
                if (klast >= kfirst) cring += ((klast + 1) >> 1) - z.cnext + 1;
                c_request<T, WXT, NIN, PRO>(p, z, kstart + n);
                // the halo vector this thread corrects: row jt-1 (threads 0 .. TC/V-1) or row jt+NR (the next TC/V threads)
                constexpr int nvr = TC / V;
                constexpr uint32_t crowb = (uint32_t)ZG<T, WXT>::template csx_v<PRO == 2> * sizeof(T);
                const int which = (int)threadIdx.x / nvr, hv = (int)threadIdx.x - which * nvr;
                const int jh = which ? jt + NR : jt - 1;
                z.h_ok = which < 2 && jh >= 1 && jh < p.sy;
                z.h_a = (uint32_t)(((which ? NR + 1 : 0) * TC + hv * V) * (int)sizeof(T));
                z.h_co = PRO == 2 ? (uint32_t)(((jh >> 1) - z.Jb) * (int)crowb + (((ct + hv * V) >> 1) - z.cbase) * (int)sizeof(T))
                                  : (uint32_t)(((jh >> 1) - z.Jb) * (int)crowb + ((hv * V) >> 1) * (int)sizeof(T));
                z.h_dj = (jh & 1) ? crowb : 0u;
                z.h_c0 = PRO == 2 ? (ct + hv * V == 0 || ct + hv * V == p.sx) : hv == 0;
            }
        }
        __syncthreads();   // coefficient table visible

        // wall / validity masks of this thread's patch
        const int jrow0 = jt + wy * ZR;                                 // grid row of patch row 0
        const int icol0 = ct + cx0;                                     // grid column of vector element 0
        z.cw0 = (icol0 == 0) || (icol0 == p.sx);
        z.wrow = jrow0 + ZR - 1 == p.sy;
        const bool col_out = p.ntx == 1 ? true : (cx0 >= V && cx0 < TC - V && icol0 < p.sx);
        z.omask = 0;
#pragma unroll
        for (int r = 0; r < ZR; ++r) {
            const int j = jrow0 + r;
            if (col_out && j >= jlo && j < jhi) z.omask |= 1 << r;
        }
        // in-plane offset of (patch row 0, element 0); halo vectors left of column 0 neither load nor store through it
        const long long own = (long long)jrow0 * p.sx + max(icol0, 0);
        z.t = kstart;
        z.kb = kb;
        z.nout = ke - kb;
        z.kend_in = kend_in;
        if (PRO) z.ce_own = (uint32_t)((((jrow0 >> 1) - z.Jb) * ZG<T, WXT>::template csx_v<PRO == 2> + ((icol0 >> 1) - (PRO == 2 ? z.cbase : 0))) * (int)sizeof(T));
        z.coef = smem_u32(coef);
        // the first z_step runs at t = kstart+1: sweep 1 makes plane kstart, sweep 2 plane kstart-1
        z.f1 = rhs + own + p.sp * kstart;
        z.o_last = out + own + p.sp * (kstart - (S - 1));

        Patch<T> X, Y, P, Q;
#pragma unroll
        for (int r = 0; r < ZR; ++r)
#pragma unroll
            for (int e = 0; e < V; ++e) X.r[r].v[e] = Y.r[r].v[e] = P.r[r].v[e] = Q.r[r].v[e] = T(0);

        const int tend = ke - 1 + S;
        z_first<T, WXT, ZERO, PRO>(p, z, tile_src, IN, X);
        // Steps come in pairs so that the loop has ONE back edge on which every register set is back in its place
        // (no moves).  An odd segment runs one idle step past its end: nothing arrives, nothing is stored (masks),
        // the coefficient table has a spare record for it.
        do {
            z_step<T, WXT, S, HAS_RHS, ZERO, NORM, PRO, ISO>(p, z, tile_src, IN, Y, X, Q, P);
            z_step<T, WXT, S, HAS_RHS, ZERO, NORM, PRO, ISO>(p, z, tile_src, IN, X, Y, P, Q);
        } while (z.t <= tend);
        // planes requested but not consumed cannot exist (requests stop at kend_in, steps run past it)
    }
    if (NORM) {
        __shared__ double s_red[16];
        double a = warp_sum(z.acc);
        if (lane == 0) s_red[warp] = a;
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
    int WX = 0, WY = 0, TC = 0, COUT = 0, ntx = 1, STEP = 0, nty = 0, ctas = 0, zcap = 0, in_plane = 0, coef_bytes = 0;
    size_t smem = 0;
    int useg = 0, nunits = 0;      // unit mode (aligned z-segments), see ZP
    int qb[ZQB];
};

// Work partition.  The work is the linearised list of (tile, plane) items, plane fastest; a CTA gets a contiguous range
// and runs one z-segment per tile it touches.  A segment of n output planes costs n + W plane steps (W: the S warm-up and
// S drain planes of the pipeline, the first step, the coefficient table and the first wait for the input ring), so equal
// ITEM counts are not equal work: a range that straddles a tile boundary pays W twice (measured at 257^3, 148 CTAs: the
// slowest SM was busy 113 k cycles against 98 k on average, and the 17 straddlers were the slow ones).  The ranges are
// cut greedily for the smallest maximum COST instead: returns the largest range length.
static int zpartition(int ntiles, int NP, int W, int ctas, int* qb)
{
    const long long N = (long long)ntiles * NP;
    auto cut = [&](long long T, int* out) -> int {     // CTAs needed when none may cost more than T
        long long q = 0;
        int n = 0;
        while (q < N) {
            if (out && n <= ctas) out[n] = (int)q;
            long long budget = T;
            while (budget > W && q < N) {                // a segment: W + at least one plane
                const long long tile_end = (q / NP + 1) * NP;
                const long long take = std::min(budget - W, tile_end - q);
                q += take;
                budget -= take + W;
            }
            if (++n > ctas && !out) return n;
        }
        if (out)
            for (int i = n; i <= ctas; ++i) out[i] = (int)N;
        return n;
    };
    long long lo = W + 1, hi = N + (long long)W * ntiles;   // cut(hi) == 1
    while (lo < hi) {
        const long long mid = (lo + hi) / 2;
        if (cut(mid, nullptr) <= ctas) hi = mid; else lo = mid + 1;
    }
    cut(lo, qb);
    int longest = 0;
    for (int i = 0; i < ctas; ++i) longest = std::max(longest, qb[i + 1] - qb[i]);
    return longest;
}

template <typename T>
static ZCfg zcfg_make(const mhs_ctx* c, const Level& lv, int S, bool zero, bool pro);

// The launch shape is a function of the level's extents, the element type, S, the variant and the SM count: computed once
// per process and kept (the partition is a small search, and zcfg is asked several times per cycle).
template <typename T>
static const ZCfg& zcfg(const mhs_ctx* c, const Level& lv, int S, bool zero, bool pro = false)
{
    using Key = std::tuple<int, int, int, int, int, int, int, int, int>;
    static std::map<Key, ZCfg> cache;
    static std::mutex mu;
    const Key key(lv.dim, lv.nx, lv.ny, lv.nz, (int)sizeof(T), S, (int)zero + 2 * (int)pro, c->num_sms, (int)lv.coarsest);
    std::lock_guard<std::mutex> lock(mu);
    auto it = cache.find(key);
    if (it == cache.end()) it = cache.emplace(key, zcfg_make<T>(c, lv, S, zero, pro)).first;
    return it->second;
}

template <typename T>
static ZCfg zcfg_make(const mhs_ctx* c, const Level& lv, int S, bool zero, bool pro)
{
    constexpr int V = ZV<T>::N;
    constexpr int NCO = ZV<T>::NCO;
    constexpr int ZR = ZV<T>::R, ZWY = ZV<T>::WY;
    ZCfg z;
    if (lv.dim != 3 || lv.coarsest || lv.nz < 5) return z;
    const int lane_cols = 32 * V;
    if (lv.sx % lane_cols != 0) return z;
    const int wfull = lv.sx / lane_cols;
    z.WY = ZWY;
    const int NR = z.WY * ZR;
    if (lv.sy < NR + 1) return z;
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
    // tiles along y: tile ty has its patch rows at 1 + ty*STEP (the last one is pulled back to end at the wall)
    z.STEP = NR - 2 * (S - 1);
    z.nty = lv.sy - NR - 1 <= 0 ? 1 : (lv.sy - NR - 1 + z.STEP - 1) / z.STEP + 1;
    const long long items = (long long)z.ntx * z.nty * (lv.nz - 2);
    if (items >= (1ll << 31)) return z;
    // one CTA per SM; a z-segment should be long against its S warm-up planes
    z.ctas = (int)std::max<long long>(1, std::min<long long>(std::min(c->num_sms, ZQB - 1), items / 12));
    // Aligned segments.  When every tile can be cut into the SAME z-segments (tiles x segments CTAs, each one segment), the
    // CTAs of y-neighbouring tiles walk the same planes at the same time and the halo rows they share are read from DRAM
    // once -- the second reader hits the L2.  Measured at 257^3 (19 tiles): 133 CTAs = 19 x 7 against 148 cost-balanced
    // ranges: 147 MB read instead of 191 MB, plain pass 57.6 -> 51.1 us although every CTA runs 42 steps instead of 39 and
    // 15 SMs idle; 114 CTAs = 19 x 6: 58.4 us.  The prolongation-fused pass is bound by issue, not by DRAM, and loses
    // (78.4 -> 80.1 us): it keeps the cost-balanced ranges over all SMs.
    // More tiles than SMs (513^3: 111): the same idea in rounds -- tiles x segments units, a multiple of the CTA count, CTA b
    // takes the units b, b + CTAs, ...; the units of one round are consecutive tiles of one z-slab (unit mode of the kernel).
    // The segment count is the one with the least plane steps per CTA.  Measured at 513^3 (111 tiles x 4 segments = 3 rounds of
    // 148): 478 -> 442 us per 2-sweep pass, 291.7 -> 304.6 V-cycles/s.
    int longest = 0;
    z.useg = 0; z.nunits = 0;
    if (!pro && !c->no_align) {
        const int ntiles = z.ntx * z.nty, NP = lv.nz - 2, W = 2 * S + 2;
        long long best_cost = -1;
        int best_seg = 0, best_ctas = 0;
        for (int seg = 1; seg <= NP / 16; ++seg) {
            const long long units = (long long)ntiles * seg;
            const int rounds = (int)((units + z.ctas - 1) / z.ctas);
            const int ctas = (int)((units + rounds - 1) / rounds);
            if (ctas * 100 < 85 * z.ctas) continue;                     // too many idle SMs
            if (sizeof(T) == 4 && rounds > 1) continue;                 // (fp32 passes are bound by issue: measured 1 % slower in rounds)
            const long long cost = (long long)rounds * ((NP + seg - 1) / seg + W);
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_seg = seg; best_ctas = ctas; }
        }
        // against the cost-balanced ranges: NP * ntiles / CTAs planes + ~1.5 warm-ups; aligned reads pay for ~12 % more steps
        const long long flat = ((long long)NP * ntiles + z.ctas - 1) / z.ctas + (3 * W) / 2;
        if (best_seg > 0 && best_cost * 100 <= flat * 112) {
            z.useg = best_seg; z.nunits = ntiles * best_seg; z.ctas = best_ctas;
            longest = (NP + best_seg - 1) / best_seg;
        }
    }
    if (!z.useg) longest = zpartition(z.ntx * z.nty, lv.nz - 2, 2 * S + 2, z.ctas, z.qb);
    z.zcap = (int)std::min<long long>(lv.nz + 1, (long long)longest + 2 * S + 3);
    z.coef_bytes = (int)(((size_t)(z.zcap + 1) * NCO * sizeof(T) + 127) / 128 * 128);
    z.in_plane = (NR + 2) * z.TC;
    const size_t plane = (size_t)z.in_plane * sizeof(T);
    const size_t limit = 227 * 1024 - 256;   // the kernel also has a little static shared memory
    z.smem = 128 + z.coef_bytes + (zero ? 0 : (pro ? 3 : ZNIN) * plane) + 2 * plane;
    if (pro) {   // the coarse rows under a tile: a ring of ZNCE coarse planes of NR/2 + 2 rows
        if (zero) return z;
        const size_t cpad = 16 / sizeof(T);
        z.smem += (size_t)ZNCE * (z.ntx == 1 ? (NR / 2 + 2) * (z.TC / 2) + cpad : (NR / 2 + 2) * (z.TC / 2 + cpad)) * sizeof(T);
    }
    if (z.smem > limit) return z;
    z.ok = true;
    return z;
}

template <typename T, int WXT, int S, bool HAS_RHS, bool ZERO, bool NORM, int PRO = 0, bool ISO = false>
static int zsweep_launch_w(mhs_ctx* c, const Level& lv, const ZCfg& z, const void* u, const void* rhs, void* out, const int* done,
                           const void* ec = nullptr, long long csp = 0)
{
    // the isotropic specialisation exists for the fp64 passes of the finest level (no right-hand side), where the time goes
    if constexpr (!ISO && !HAS_RHS && !ZERO && sizeof(T) == 8) {
        if (lv.hx == lv.hy) return zsweep_launch_w<T, WXT, S, HAS_RHS, ZERO, NORM, PRO, true>(c, lv, z, u, rhs, out, done, ec, csp);
    }
    auto kern = k_zsweep<T, WXT, S, HAS_RHS, ZERO, NORM, PRO, ISO>;
    static PerDevice attr;
    per_device(attr, c, [&] {
        cudaFuncAttributes fa;
        size_t stat = 4096;
        if (cudaFuncGetAttributes(&fa, kern) == cudaSuccess) stat = fa.sharedSizeBytes;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024 - stat));
        return 1;
    });
    ZP<T> p;
    p.sx = lv.sx; p.sy = lv.sy; p.nz = lv.nz; p.sp = lv.sp;
    p.tab = (const T*)lv.tab;
    p.cz = (T)(1.0 / (lv.hz * lv.hz));
    p.a2 = (T)(c->alpha * c->alpha);
    p.rho = (T)((lv.hy * lv.hy) / (lv.hx * lv.hx));
    p.WX = z.WX; p.WY = z.WY; p.TC = z.TC; p.COUT = z.COUT; p.ntx = z.ntx; p.STEP = z.STEP; p.nty = z.nty;
    p.NP = lv.nz - 2;
    p.items = (long long)z.ntx * z.nty * p.NP;
    p.zcap = z.zcap;
    p.in_plane = z.in_plane;
    p.coef_bytes = z.coef_bytes;
    p.ec = (const T*)ec; p.csp = csp;
    p.useg = z.useg; p.nunits = z.nunits;
    if (!z.useg)
        for (int i = 0; i <= z.ctas; ++i) p.qb[i] = z.qb[i];
    else
        p.qb[0] = p.qb[1] = 0;
    if (z.ntx > 1) c->prof.xtiled_zsweep += 1;
    launch_pdl(c, kern, dim3(z.ctas), dim3(WXT * ZV<T>::WY * 32), z.smem, p, (const T*)u, (const T*)rhs, (T*)out, c->partial, done);
    if (c->debug) {
        cudaError_t e = cudaPeekAtLastError();
        fprintf(stderr, "[mhs] k_zsweep<%s,WX=%d,S=%d,rhs=%d,zero=%d,norm=%d,pro=%d,iso=%d> %dx%dx%d TC %d ntx %d nty %d ctas %d smem %zu: %s\n",
                sizeof(T) == 8 ? "f64" : "f32", WXT, S, (int)HAS_RHS, (int)ZERO, (int)NORM, (int)PRO, (int)ISO, lv.nx, lv.ny, lv.nz, z.TC, z.ntx, z.nty,
                z.ctas, z.smem, cudaGetErrorString(e));
    }
    return z.ctas;
}

template <typename T, int S, bool HAS_RHS, bool ZERO, bool NORM>
static int zsweep_launch(mhs_ctx* c, const Level& lv, const ZCfg& z, const void* u, const void* rhs, void* out, const int* done)
{
    switch (z.WX) {
        case 1: return zsweep_launch_w<T, 1, S, HAS_RHS, ZERO, NORM>(c, lv, z, u, rhs, out, done);
        case 2: return zsweep_launch_w<T, 2, S, HAS_RHS, ZERO, NORM>(c, lv, z, u, rhs, out, done);
        case 3: return zsweep_launch_w<T, 3, S, HAS_RHS, ZERO, NORM>(c, lv, z, u, rhs, out, done);
        default: return zsweep_launch_w<T, 4, S, HAS_RHS, ZERO, NORM>(c, lv, z, u, rhs, out, done);
    }
}

template <typename T, int S, bool HAS_RHS>
static void zsweep_launch_pro(mhs_ctx* c, const Level& lv, const ZCfg& z, const void* u, const void* rhs, void* out, const int* done,
                              const void* ec, long long csp)
{
    if (z.ntx > 1) {     // x-tiles (3 or 4 warps wide): the variant whose coarse rows come in row by row (PRO = 2)
        if (z.WX == 3) zsweep_launch_w<T, 3, S, HAS_RHS, false, false, 2>(c, lv, z, u, rhs, out, done, ec, csp);
        else zsweep_launch_w<T, 4, S, HAS_RHS, false, false, 2>(c, lv, z, u, rhs, out, done, ec, csp);
        return;
    }
    switch (z.WX) {
        case 1: zsweep_launch_w<T, 1, S, HAS_RHS, false, false, 1>(c, lv, z, u, rhs, out, done, ec, csp); break;
        case 2: zsweep_launch_w<T, 2, S, HAS_RHS, false, false, 1>(c, lv, z, u, rhs, out, done, ec, csp); break;
        case 3: zsweep_launch_w<T, 3, S, HAS_RHS, false, false, 1>(c, lv, z, u, rhs, out, done, ec, csp); break;
        default: zsweep_launch_w<T, 4, S, HAS_RHS, false, false, 1>(c, lv, z, u, rhs, out, done, ec, csp); break;
    }
}

// S (1 or 2) sweeps of level lv applied to u + P e_c (e_c = co's iterate `ec`): the trilinear correction is folded into the
// pass, u itself is not modified.  Returns false (nothing launched) when the level cannot run in k_zsweep at all.
bool launch_zsweep_prolong(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int S, const Level& co, const void* ec,
                           const int* done)
{
    if (co.sx * 2 != lv.sx) return false;
    if (c->es == 8) {
        const ZCfg& z = zcfg<double>(c, lv, S, false, true);
        if (!z.ok) return false;
        count_launch(c);
        if (rhs) { if (S == 2) zsweep_launch_pro<double, 2, true>(c, lv, z, u, rhs, out, done, ec, co.sp); else zsweep_launch_pro<double, 1, true>(c, lv, z, u, rhs, out, done, ec, co.sp); }
        else { if (S == 2) zsweep_launch_pro<double, 2, false>(c, lv, z, u, rhs, out, done, ec, co.sp); else zsweep_launch_pro<double, 1, false>(c, lv, z, u, rhs, out, done, ec, co.sp); }
    } else {
        const ZCfg& z = zcfg<float>(c, lv, S, false, true);
        if (!z.ok) return false;
        count_launch(c);
        if (rhs) { if (S == 2) zsweep_launch_pro<float, 2, true>(c, lv, z, u, rhs, out, done, ec, co.sp); else zsweep_launch_pro<float, 1, true>(c, lv, z, u, rhs, out, done, ec, co.sp); }
        else { if (S == 2) zsweep_launch_pro<float, 2, false>(c, lv, z, u, rhs, out, done, ec, co.sp); else zsweep_launch_pro<float, 1, false>(c, lv, z, u, rhs, out, done, ec, co.sp); }
    }
    return true;
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
        const ZCfg& z = zcfg<T>(c, lv, SS, ZERO);                                         \
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
