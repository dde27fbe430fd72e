// The small-level kernel of libmhs_b200: ONE launch runs the whole lower part of the V-cycle -- every level
// from the first one that is too small to fill the GPU down to the exact coarsest solve and back up -- on ONE
// thread-block cluster, with hardware cluster barriers between the multigrid phases instead of kernel launches.
//
//   * "cluster levels" (a few hundred thousand nodes at most: they live in the L2) are worked on by all CTAs of
//     the cluster out of global memory, one warp per row segment; a phase (sweep, residual, restriction,
//     prolongation) ends in cluster.sync(), a ~0.2 us hardware barrier that also orders global memory.
//   * "tail levels" (everything that fits in one SM's shared memory: u, rhs and a scratch array per level)
//     are done by CTA 0 alone with __syncthreads() between the phases.
//   * When the FINEST level of a hierarchy is itself a cluster level (the 2D boundary problem up to 513^2, the
//     33^3 configuration) the kernel runs the whole SOLVE: residual norm, stop rule, V-cycle, repeated on the
//     device until the stop rule fires -- one launch per mhs_solve_* call, no host round trip per cycle.
//
// On these levels the work is tiny and the paper's one-kernel-per-function design pays launch
// latency ~25 times per level pair; this is what removes it.  Arithmetic: the same formulas as the reference
// kernels (mhs_device.cuh), so the iterates are identical up to the order of the norm's summation.
#include <cooperative_groups.h>

#include <cstdio>
#include <cstdlib>

#include "mhs_device.cuh"

namespace cg = cooperative_groups;

namespace mhs {

constexpr int CL_THREADS = 1024;
constexpr int CL_MAXG = 4;             // cluster levels per launch
constexpr long long CL_MAX_PTS = 600000;  // largest level given to the cluster instead of the whole GPU

template <typename T>
struct TailLevelP {
    int nx, ny, nz;
    int bx, by;                   // bits of the power-of-two index space of the interior nodes along x, y
    int off_u, off_rhs, off_tmp;  // element offsets into the shared array
    int off_tab;                  // shared copy of the level's table cx | cy | diag | w (4 nz entries); -1: none, read `tab`
    const T* tab;                 // global: cx | cy | diag | w
    T cz;
};

template <typename T>
struct GLevelP {                  // a cluster level: aliased Dirichlet layout in global memory
    int nx, ny, nz, sx, sy, sp;
    const T* tab;
    T cz;
    T *u, *tmp, *rhs, *r;         // rhs == nullptr: zero right-hand side (finest 3D level)
};

template <typename T>
struct ClusterP {
    int mode;                     // 0: V pass from level g[0] with zero initial guess; 1: one V-cycle continuing
                                  // from g[0].u; 2: solve loop (norm, stop rule, V-cycle) on g[0]
    int nglob, ntail, dim3, n_pre, n_post, ncoarse;
    T a2;
    GLevelP<T> g[CL_MAXG];
    TailLevelP<T> t[8];
    const T* ainv;                // global, ncoarse^2 (coarsest level, exact inverse)
    int tail_tot;                 // elements of the tail's level arrays (zeroed at the start)
    int off_ainv;                 // shared copy of ainv (-1: it did not fit, read from global)
    const T* tail_rhs_g;          // top tail level, aliased layout (in)
    T* tail_u_g;                  // top tail level, aliased layout (out)
    int tail_sx, tail_sp;
    double* partial;              // >= cluster size doubles
    Ctl* ctl;
};

template <typename T>
__device__ __forceinline__ T ldcg(const T* p) { return __ldcg(p); }

// -DMHS_TAILPROF (a tuning build, never the shipped one): thread 0 of CTA 0 stamps clock64() after every phase of one
// cycle; mhs_debug_tailprof() reads the stamps back.
#ifdef MHS_TAILPROF
__device__ long long g_tp[2 * 512];
__device__ int g_tpn, g_tp_on;
#define TP(id)                                                                      \
    do {                                                                            \
        if (threadIdx.x == 0 && blockIdx.x == 0 && g_tp_on && g_tpn < 512) {        \
            g_tp[2 * g_tpn] = (id); g_tp[2 * g_tpn + 1] = clock64(); ++g_tpn;       \
        }                                                                           \
    } while (0)
// a solve loop (mode 2) keeps the stamps of its second cycle, a single V pass those of the launch
#define TP_RESET(cyc, mode2)                                                        \
    do {                                                                            \
        if (threadIdx.x == 0 && blockIdx.x == 0) {                                  \
            g_tp_on = !(mode2) || (cyc) == 1;                                       \
            if (g_tp_on) g_tpn = 0;                                                 \
        }                                                                           \
    } while (0)
#else
#define TP(id) do { } while (0)
#define TP_RESET(cyc, mode2) do { } while (0)
#endif

// ---------------------------------------------------------------------------------------------
// tail: levels in shared memory, plain dense layout (nx*ny*nz, walls stored as zeros), CTA 0 only
// ---------------------------------------------------------------------------------------------
// Interior nodes of a tail level are enumerated through a power-of-two index space (bx, by, bz bits per axis), so
// that a thread turns its work index into (i, j, k) with shifts and masks instead of integer divisions.
template <typename T>
struct TailIdx {
    int mx, my, k0, k1, bx, bxy, n, nx, nxy;
    __device__ __forceinline__ TailIdx(const TailLevelP<T>& L, bool d3)
        : mx(L.nx - 2), my(L.ny - 2), k0(d3 ? 1 : 0), k1(d3 ? L.nz - 1 : 1), bx(L.bx), bxy(L.bx + L.by), nx(L.nx), nxy(L.nx * L.ny)
    {
        n = (k1 - k0) << bxy;
    }
    __device__ __forceinline__ bool at(int q, int& i, int& j, int& k, int& c) const
    {
        i = (q & ((1 << bx) - 1)) + 1;
        j = ((q >> bx) & ((1 << (bxy - bx)) - 1)) + 1;
        k = (q >> bxy) + k0;
        c = i + nx * j + nxy * k;
        return i <= mx && j <= my;
    }
    __device__ __forceinline__ bool at(int q, int& k, int& c) const
    {
        int i, j;
        return at(q, i, j, k, c);
    }
};

template <typename T, bool d3>
__device__ __forceinline__ T tail_Lu(const TailLevelP<T>& L, const T* tab, const T* u, int c, int k, T a2)
{
    const int nx = L.nx, nxy = L.nx * L.ny;
    const T uc = u[c];
    T lu = tab[k] * lap1<T>(u[c + 1], u[c - 1], uc) + tab[L.nz + k] * lap1<T>(u[c + nx], u[c - nx], uc);
    if (d3) lu += L.cz * lap1<T>(u[c + nxy], u[c - nxy], uc) + a2 * uc;
    return lu;
}

// dst = src + (omega/D_k)(rhs - L src) at the interior nodes (a2)
template <typename T, bool d3>
__device__ __forceinline__ void tail_sweep(const TailLevelP<T>& L, const T* tab, const T* src, T* dst, const T* rhs, T a2)
{
    const TailIdx<T> I(L, d3);
    for (int q = threadIdx.x; q < I.n; q += blockDim.x) {
        int k, c;
        if (I.at(q, k, c)) dst[c] = src[c] + tab[3 * L.nz + k] * (rhs[c] - tail_Lu<T, d3>(L, tab, src, c, k, a2));
    }
    __syncthreads();
}

// The first TWO sweeps from the zero initial guess in one phase: sweep 1 is u1 = (omega/D_k) rhs (rhs is zero on
// every wall, so u1 is too), formed on the fly at the seven nodes sweep 2 reads.
template <typename T, bool d3>
__device__ __forceinline__ void tail_sweep2_from_zero(const TailLevelP<T>& L, const T* tab, T* dst, const T* rhs, T a2)
{
    const TailIdx<T> I(L, d3);
    const int nx = L.nx, nxy = L.nx * L.ny;
    for (int q = threadIdx.x; q < I.n; q += blockDim.x) {
        int k, c;
        if (!I.at(q, k, c)) continue;
        const T w = tab[3 * L.nz + k];
        const T f = rhs[c], uc = w * f;
        T lu = tab[k] * lap1<T>(w * rhs[c + 1], w * rhs[c - 1], uc) + tab[L.nz + k] * lap1<T>(w * rhs[c + nx], w * rhs[c - nx], uc);
        if (d3) lu += L.cz * lap1<T>(tab[3 * L.nz + k + 1] * rhs[c + nxy], tab[3 * L.nz + k - 1] * rhs[c - nxy], uc) + a2 * uc;
        dst[c] = uc + w * (f - lu);
    }
    __syncthreads();
}

// What does not depend on earlier kernels, done BEFORE the kernel waits for them (pdl_wait): the level arrays zeroed
// (walls must read as zeros), the coefficient tables and the coarsest inverse copied into shared memory.  Measured on the
// 3D tail (one launch per cycle): the first touch of every level's table and of ainv was an L2 miss of ~1 us each.
template <typename T>
__device__ __forceinline__ void tail_zero(const ClusterP<T>& P, T* S)
{
    for (int q = threadIdx.x; q < P.tail_tot; q += blockDim.x) S[q] = T(0);
}

template <typename T>
__device__ void tail_prologue(const ClusterP<T>& P, T* S)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    tail_zero<T>(P, S);
    for (int l = 0; l < P.ntail; ++l) {
        const TailLevelP<T>& L = P.t[l];
        if (L.off_tab >= 0)
            for (int q = tid; q < 4 * L.nz; q += nt) S[L.off_tab + q] = L.tab[q];
    }
    if (P.off_ainv >= 0)
        for (int q = tid; q < P.ncoarse * P.ncoarse; q += nt) S[P.off_ainv + q] = P.ainv[q];
    // (the first __syncthreads of tail_body orders these stores before their use)
}

template <typename T, bool d3>
__device__ void tail_body(const ClusterP<T>& P, T* S)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    const int nlev = P.ntail;
    T* cur[8];   // which of a level's two iterate buffers holds its iterate (they ping-pong)
    T* oth[8];

    // load the top level's right-hand side (everything else is zero: tail_prologue / tail_zero)
    {
        const TailLevelP<T>& L = P.t[0];
        const TailIdx<T> I(L, d3);
        for (int q = tid; q < I.n; q += nt) {
            int i, j, k, c;
            if (!I.at(q, i, j, k, c)) continue;
            S[L.off_rhs + c] = ldcg(P.tail_rhs_g + i + P.tail_sx * j + P.tail_sp * k);
        }
    }
    __syncthreads();
    TP(100);

    // ---- down leg ----
    for (int l = 0; l < nlev - 1; ++l) {
        const TailLevelP<T>& L = P.t[l];
        const TailLevelP<T>& C = P.t[l + 1];
        const T* tab = L.off_tab >= 0 ? S + L.off_tab : L.tab;
        cur[l] = S + L.off_u;
        oth[l] = S + L.off_tmp;
        const T* rhs = S + L.off_rhs;
        int s0 = 0;
        if (P.n_pre >= 2) {
            tail_sweep2_from_zero<T, d3>(L, tab, cur[l], rhs, P.a2);
            s0 = 2;
            TP(1000 * (l + 1) + 1);
        }
        for (int s = s0; s < P.n_pre; ++s) {   // (n_pre == 1: one ordinary sweep from the zero-filled buffer)
            tail_sweep<T, d3>(L, tab, cur[l], oth[l], rhs, P.a2);
            T* x = cur[l]; cur[l] = oth[l]; oth[l] = x;
        }
        // residual -> the free iterate buffer (its walls are never read by the weighting below)
        T* r = oth[l];
        {
            const TailIdx<T> I(L, d3);
            for (int q = tid; q < I.n; q += nt) {
                int k, c;
                if (I.at(q, k, c)) r[c] = rhs[c] - tail_Lu<T, d3>(L, tab, cur[l], c, k, P.a2);
            }
        }
        __syncthreads();
        TP(1000 * (l + 1) + 2);
        // full weighting -> rhs of the next level
        {
            const TailIdx<T> I(C, d3);
            T* rc = S + C.off_rhs;
            for (int q = tid; q < I.n; q += nt) {
                int Ii, J, K, cc;
                if (!I.at(q, Ii, J, K, cc)) continue;
                const T* r0 = r + 2 * Ii + L.nx * (2 * J) + L.nx * L.ny * (2 * K);
                T s = T(0);
#pragma unroll
                for (int dc = (d3 ? -1 : 0); dc <= (d3 ? 1 : 0); ++dc) {
                    T sp = T(0);
#pragma unroll
                    for (int db = -1; db <= 1; ++db) {
                        const T* row = r0 + L.nx * db + L.nx * L.ny * dc;
                        const T sxv = T(0.25) * (row[-1] + row[1]) + T(0.5) * row[0];
                        sp += (db == 0 ? T(0.5) : T(0.25)) * sxv;
                    }
                    s += (d3 ? (dc == 0 ? T(0.5) : T(0.25)) : T(1)) * sp;
                }
                rc[cc] = s;
            }
        }
        __syncthreads();
        TP(1000 * (l + 1) + 3);
        // the residual's buffer goes back to being an iterate buffer: its interior is overwritten before it is read
    }

    // ---- coarsest level: exact solve e = A^-1 rhs (C9) ----
    {
        const TailLevelP<T>& L = P.t[nlev - 1];
        const int mx = L.nx - 2, my = L.ny - 2, k0 = d3 ? 1 : 0;
        const int n = P.ncoarse;
        T* u = S + L.off_u;
        cur[nlev - 1] = u;
        const T* rhs = S + L.off_rhs;
        T* cr = S + L.off_tmp;   // the coarsest level's scratch array: its right-hand side as a dense vector
        const T* ainv = P.off_ainv >= 0 ? S + P.off_ainv : P.ainv;
        auto cell = [&](int row) {
            const int i = row % mx, j = (row / mx) % my, k = row / (mx * my);
            return (i + 1) + L.nx * (j + 1) + L.nx * L.ny * (k + k0);
        };
        for (int row = tid; row < n; row += nt) cr[row] = rhs[cell(row)];
        __syncthreads();
        for (int row = tid; row < n; row += nt) {
            double s = 0.0;
            for (int col = 0; col < n; ++col) s += (double)ainv[(long long)row * n + col] * (double)cr[col];
            u[cell(row)] = (T)s;
        }
        __syncthreads();
        TP(1000 * nlev + 4);
    }

    // ---- up leg ----
    for (int l = nlev - 2; l >= 0; --l) {
        const TailLevelP<T>& L = P.t[l];
        const TailLevelP<T>& C = P.t[l + 1];
        const T* tab = L.off_tab >= 0 ? S + L.off_tab : L.tab;
        const T* rhs = S + L.off_rhs;
        const T* ec = cur[l + 1];
        {
            const TailIdx<T> I(L, d3);
            T* u = cur[l];
            const int cxy = C.nx * C.ny;
            for (int q = tid; q < I.n; q += nt) {
                int i, j, k, c;
                if (!I.at(q, i, j, k, c)) continue;
                const int I0 = i >> 1, I1 = (i + 1) >> 1, J0 = j >> 1, J1 = (j + 1) >> 1, K0 = k >> 1, K1 = (k + 1) >> 1;
                T s = (ec[I0 + C.nx * J0 + cxy * K0] + ec[I1 + C.nx * J0 + cxy * K0]) +
                      (ec[I0 + C.nx * J1 + cxy * K0] + ec[I1 + C.nx * J1 + cxy * K0]);
                if (d3)
                    s += (ec[I0 + C.nx * J0 + cxy * K1] + ec[I1 + C.nx * J0 + cxy * K1]) +
                         (ec[I0 + C.nx * J1 + cxy * K1] + ec[I1 + C.nx * J1 + cxy * K1]);
                u[c] += (d3 ? T(0.125) : T(0.25)) * s;
            }
        }
        __syncthreads();
        TP(1000 * (l + 1) + 5);
        for (int s = 0; s < P.n_post; ++s) {
            tail_sweep<T, d3>(L, tab, cur[l], oth[l], rhs, P.a2);
            T* x = cur[l]; cur[l] = oth[l]; oth[l] = x;
            TP(1000 * (l + 1) + 6 + s);
        }
    }

    // ---- write the correction of the top tail level back (interior nodes) ----
    {
        const TailLevelP<T>& L = P.t[0];
        const TailIdx<T> I(L, d3);
        const T* u = cur[0];
        for (int q = tid; q < I.n; q += nt) {
            int i, j, k, c;
            if (!I.at(q, i, j, k, c)) continue;
            P.tail_u_g[i + P.tail_sx * j + P.tail_sp * k] = u[c];
        }
    }
    TP(101);
}

// ---------------------------------------------------------------------------------------------
// cluster levels: phases over global memory.  Work item = 32 consecutive interior nodes of one row;
// items are dealt round-robin to all warps of the cluster.  Loads go through ld.global.cg: what one
// CTA wrote in the previous phase must be seen by the others (L1 is not coherent across SMs).
// ---------------------------------------------------------------------------------------------
struct Who { int wg, nW, lane; };

template <typename T, bool D3>
struct RowIt {     // iterates the interior row segments of a level
    int xch, nitems, sy1, xsh;   // xsh: log2(xch) when the number of 32-node segments per row is a power of two (a shift instead of a division)
    __device__ RowIt(int sx, int sy, int nz) : xch((sx - 1 + 31) / 32), sy1(sy - 1)
    {
        nitems = sy1 * (D3 ? nz - 2 : 1) * xch;
        xsh = (xch & (xch - 1)) == 0 ? __ffs(xch) - 1 : -1;
    }
    __device__ __forceinline__ bool at(int it, int lane, int sx, int sp, int& i, int& j, int& k, int& idx) const
    {
        const int row = xsh >= 0 ? it >> xsh : it / xch, c = it - row * xch;
        const int kk = D3 ? row / sy1 : 0, jj = row - kk * sy1;
        i = 1 + 32 * c + lane; j = jj + 1; k = D3 ? kk + 1 : 0;
        idx = i + sx * j + sp * k;
        return i < sx;
    }
};

template <typename T, bool D3>
__device__ __forceinline__ T g_Lu(const GLevelP<T>& L, const T* __restrict__ u, int idx, int k, T a2)
{
    const T uc = ldcg(u + idx);
    T lu = L.tab[k] * lap1<T>(ldcg(u + idx + 1), ldcg(u + idx - 1), uc) +
           L.tab[L.nz + k] * lap1<T>(ldcg(u + idx + L.sx), ldcg(u + idx - L.sx), uc);
    if (D3) lu += L.cz * lap1<T>(ldcg(u + idx + L.sp), ldcg(u + idx - L.sp), uc) + a2 * uc;
    return lu;
}

// out = u + (omega/D_k) (rhs - L u)     (a2).  NORM: also this thread's sum of (rhs - L u)^2, the squared
// residual of the INPUT iterate (a7) -- the sweep forms that residual anyway, so the stop test costs no phase of its own.
template <typename T, bool D3, bool NORM>
__device__ double ph_sweep(const GLevelP<T>& L, const T* __restrict__ u, const T* __restrict__ rhs, T* __restrict__ out, T a2, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
    double acc = 0.0;
    if (!D3) {   // one plane: the coefficients are three numbers, read once per phase instead of once per item
        const T cx = L.tab[0], cy = L.tab[L.nz], wk = L.tab[3 * L.nz];
#pragma unroll 4
        for (int it = w.wg; it < R.nitems; it += w.nW) {
            int i, j, k, idx;
            if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
            const T f = rhs ? ldcg(rhs + idx) : T(0);
            const T uc = ldcg(u + idx);
            const T r = f - (cx * lap1<T>(ldcg(u + idx + 1), ldcg(u + idx - 1), uc) + cy * lap1<T>(ldcg(u + idx + L.sx), ldcg(u + idx - L.sx), uc));
            out[idx] = uc + wk * r;
            if (NORM) acc += (double)r * (double)r;
        }
        return acc;
    }
#pragma unroll 4
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        const T f = rhs ? ldcg(rhs + idx) : T(0);
        const T r = f - g_Lu<T, D3>(L, u, idx, k, a2);
        out[idx] = ldcg(u + idx) + L.tab[3 * L.nz + k] * r;
        if (NORM) acc += (double)r * (double)r;
    }
    return acc;
}

// The first TWO sweeps from the zero initial guess in one phase: sweep 1 is u1 = (omega/D_k) rhs (rhs is zero on every
// wall, so u1 is too), formed on the fly at the nodes sweep 2 reads (as tail_sweep2_from_zero).
template <typename T, bool D3>
__device__ void ph_sweep2_zero(const GLevelP<T>& L, const T* __restrict__ rhs, T* __restrict__ out, T a2, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
#pragma unroll 2
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        const T wk = L.tab[3 * L.nz + k];
        const T f = ldcg(rhs + idx), uc = wk * f;
        T lu = L.tab[k] * lap1<T>(wk * ldcg(rhs + idx + 1), wk * ldcg(rhs + idx - 1), uc) +
               L.tab[L.nz + k] * lap1<T>(wk * ldcg(rhs + idx + L.sx), wk * ldcg(rhs + idx - L.sx), uc);
        if (D3) lu += L.cz * lap1<T>(L.tab[3 * L.nz + k + 1] * ldcg(rhs + idx + L.sp), L.tab[3 * L.nz + k - 1] * ldcg(rhs + idx - L.sp), uc) + a2 * uc;
        out[idx] = uc + wk * (f - lu);
    }
}

// 2D: residual + full weighting in one phase.  The residual is formed at the nine fine nodes under a coarse node from a
// sliding window of three fine rows in registers, with the formula and the summation order of ph_residual / ph_restrict
// (the same bits); the residual array is not used.
template <typename T>
__device__ void ph_resid_restrict2(const GLevelP<T>& L, const T* __restrict__ u, const T* __restrict__ rhs, int csx, int csy, T* __restrict__ rc, Who w)
{
    const RowIt<T, false> R(csx, csy, 1);
    const T cx = L.tab[0], cy = L.tab[L.nz];
    const int fsx = L.sx;
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int I, J, K, cidx;
        if (!R.at(it, w.lane, csx, 0, I, J, K, cidx)) continue;
        const int c0 = 2 * I + fsx * (2 * J);
        T ra[3], rb[5], rn[5];    // fine rows y-1 (columns -1..1), y and y+1 (columns -2..2) around the row being reduced
#pragma unroll
        for (int a = 0; a < 3; ++a) ra[a] = ldcg(u + c0 - 2 * fsx + a - 1);
#pragma unroll
        for (int a = 0; a < 5; ++a) rb[a] = ldcg(u + c0 - fsx + a - 2);
        T sp = T(0);
#pragma unroll
        for (int db = -1; db <= 1; ++db) {
#pragma unroll
            for (int a = 0; a < 5; ++a) rn[a] = (db < 1 || (a >= 1 && a <= 3)) ? ldcg(u + c0 + (db + 1) * fsx + a - 2) : T(0);
            T r[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const T uc = rb[a + 1];
                const T lu = cx * lap1<T>(rb[a + 2], rb[a], uc) + cy * lap1<T>(rn[a + 1], ra[a], uc);
                const T f = rhs ? ldcg(rhs + c0 + db * fsx + a - 1) : T(0);
                r[a] = f - lu;
            }
            const T sxv = T(0.25) * (r[0] + r[2]) + T(0.5) * r[1];
            sp += (db == 0 ? T(0.5) : T(0.25)) * sxv;
#pragma unroll
            for (int a = 0; a < 3; ++a) ra[a] = rb[a + 1];
#pragma unroll
            for (int a = 0; a < 5; ++a) rb[a] = rn[a];
        }
        rc[cidx] = sp;
    }
}

// 2D: prolongation + correction + the first post-smoothing sweep in one phase: out = sweep(u + P e_c), the corrected
// value formed on the fly (with ph_prolong's expression) at the five nodes the sweep reads.  On a wall node the
// interpolated correction is zero by itself (coarse walls are stored zeros), so no node needs a test.
template <typename T>
__device__ void ph_prolong_sweep2(const GLevelP<T>& L, const T* __restrict__ u, const T* __restrict__ rhs, const T* __restrict__ ec, int csx,
                                  T* __restrict__ out, Who w)
{
    const RowIt<T, false> R(L.sx, L.sy, 1);
    const T cx = L.tab[0], cy = L.tab[L.nz], wk = L.tab[3 * L.nz];
    const int sx = L.sx;
    auto corrected = [&](int a, int b) -> T {
        const int I0 = a >> 1, I1 = (a + 1) >> 1, J0 = b >> 1, J1 = (b + 1) >> 1;
        const T s = (ldcg(ec + I0 + csx * J0) + ldcg(ec + I1 + csx * J0)) + (ldcg(ec + I0 + csx * J1) + ldcg(ec + I1 + csx * J1));
        return ldcg(u + a + sx * b) + T(0.25) * s;
    };
#pragma unroll 2
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, sx, 0, i, j, k, idx)) continue;
        const T uc = corrected(i, j);
        const T lu = cx * lap1<T>(corrected(i + 1, j), corrected(i - 1, j), uc) + cy * lap1<T>(corrected(i, j + 1), corrected(i, j - 1), uc);
        const T f = rhs ? ldcg(rhs + idx) : T(0);
        out[idx] = uc + wk * (f - lu);
    }
}

// first sweep from the zero initial guess: u = (omega/D_k) rhs
template <typename T, bool D3>
__device__ void ph_scale(const GLevelP<T>& L, const T* __restrict__ rhs, T* __restrict__ out, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
#pragma unroll 4
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        out[idx] = L.tab[3 * L.nz + k] * ldcg(rhs + idx);
    }
}

template <typename T, bool D3>
__device__ void ph_zero(const GLevelP<T>& L, T* __restrict__ out, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) out[idx] = T(0);
    }
}

// r = rhs - L u   (a3)
template <typename T, bool D3>
__device__ void ph_residual(const GLevelP<T>& L, const T* __restrict__ u, const T* __restrict__ rhs, T* __restrict__ r, T a2, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
#pragma unroll 4
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        const T f = rhs ? ldcg(rhs + idx) : T(0);
        r[idx] = f - g_Lu<T, D3>(L, u, idx, k, a2);
    }
}

// sum over interior nodes of (rhs - L u)^2 for this thread's items   (a7)
template <typename T, bool D3>
__device__ double ph_resnorm(const GLevelP<T>& L, const T* __restrict__ u, const T* __restrict__ rhs, T a2, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
    double acc = 0.0;
#pragma unroll 4
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        const T f = rhs ? ldcg(rhs + idx) : T(0);
        const double r = (double)(f - g_Lu<T, D3>(L, u, idx, k, a2));
        acc += r * r;
    }
    return acc;
}

// full weighting of r (fine, pitch fsx/fsp) into the coarse interior nodes   (a4)
template <typename T, bool D3>
__device__ void ph_restrict(const T* __restrict__ r, int fsx, int fsp, int csx, int csy, int cnz, int csp, T* __restrict__ rc, Who w)
{
    const RowIt<T, D3> R(csx, csy, cnz);
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int I, J, K, cidx;
        if (!R.at(it, w.lane, csx, csp, I, J, K, cidx)) continue;
        const T* q = r + 2 * I + fsx * (2 * J) + fsp * (2 * K);
        T s = T(0);
#pragma unroll
        for (int dc = (D3 ? -1 : 0); dc <= (D3 ? 1 : 0); ++dc) {
            T sp = T(0);
#pragma unroll
            for (int db = -1; db <= 1; ++db) {
                const T* row = q + fsx * db + fsp * dc;
                const T sxv = T(0.25) * (ldcg(row - 1) + ldcg(row + 1)) + T(0.5) * ldcg(row);
                sp += (db == 0 ? T(0.5) : T(0.25)) * sxv;
            }
            s += (D3 ? (dc == 0 ? T(0.5) : T(0.25)) : T(1)) * sp;
        }
        rc[cidx] = s;
    }
}

// u += P e_c  (tri/bi-linear, a6)
template <typename T, bool D3>
__device__ void ph_prolong(const GLevelP<T>& L, T* __restrict__ u, const T* __restrict__ ec, int csx, int csp, Who w)
{
    const RowIt<T, D3> R(L.sx, L.sy, L.nz);
#pragma unroll 4
    for (int it = w.wg; it < R.nitems; it += w.nW) {
        int i, j, k, idx;
        if (!R.at(it, w.lane, L.sx, L.sp, i, j, k, idx)) continue;
        const int I0 = i >> 1, I1 = (i + 1) >> 1, J0 = j >> 1, J1 = (j + 1) >> 1, K0 = k >> 1, K1 = (k + 1) >> 1;
        const T* a = ec + csp * K0;
        T s = (ldcg(a + I0 + csx * J0) + ldcg(a + I1 + csx * J0)) + (ldcg(a + I0 + csx * J1) + ldcg(a + I1 + csx * J1));
        if (D3) {
            const T* b = ec + csp * K1;
            s += (ldcg(b + I0 + csx * J0) + ldcg(b + I1 + csx * J0)) + (ldcg(b + I0 + csx * J1) + ldcg(b + I1 + csx * J1));
        }
        u[idx] = ldcg(u + idx) + (D3 ? T(0.125) : T(0.25)) * s;
    }
}

template <typename T, bool D3>
__global__ void __launch_bounds__(CL_THREADS, 1) k_cluster(const __grid_constant__ ClusterP<T> P, const int* __restrict__ done)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* S = reinterpret_cast<T*>(smem_raw);
    // mode 2: every CTA keeps a copy of the control block and applies the stop rule to it itself (same inputs, same
    // decision: no second barrier to hand the decision round); CTA 0 writes its copy back at the end.
    __shared__ Ctl s_ctl;
    __shared__ int s_stop;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), ncta = (int)cluster.num_blocks();
    pdl_launch_dependents();
    if (rank == 0 && P.ntail > 0) tail_prologue<T>(P, S);   // nothing in it depends on earlier kernels
    pdl_wait();
    if (P.mode != 2 && done && *done) return;
    Who w;
    w.lane = threadIdx.x & 31;
    w.wg = (threadIdx.x >> 5) * ncta + rank;   // interleave the CTAs: consecutive row segments go to different SMs
    w.nW = ncta * (CL_THREADS / 32);
    const int ng = P.nglob;
    if (P.mode == 2) {
        const int* src = reinterpret_cast<const int*>(P.ctl);
        int* dst = reinterpret_cast<int*>(&s_ctl);
        for (int q = threadIdx.x; q < (int)(sizeof(Ctl) / sizeof(int)); q += CL_THREADS) dst[q] = __ldcg(src + q);
        __syncthreads();
    }

    // current location of each cluster level's iterate (ping-pong)
    T* cu[CL_MAXG];
    T* ct[CL_MAXG];
#pragma unroll
    for (int l = 0; l < CL_MAXG; ++l) { cu[l] = P.g[l].u; ct[l] = P.g[l].tmp; }

    // Residual norm -> stop rule (a7; C10).  acc: this thread's share of the squared norm.  One cluster barrier; true = stop.
    // The partial sums alternate between two halves of P.partial: a CTA may already be writing the next cycle's sum while
    // another still reads this cycle's.
    int flip = 0;
    auto stop_phase = [&](double acc) -> bool {
        acc = block_sum<CL_THREADS>(acc);
        double* part = P.partial + 16 * flip;
        flip ^= 1;
        if (threadIdx.x == 0) part[rank] = acc;
        cluster.sync();
        if (threadIdx.x == 0) {
            double v = 0.0;
            for (int q = 0; q < ncta; ++q) v += __ldcg(part + q);
            stop_rule(&s_ctl, sqrt(v), 1);
            s_stop = s_ctl.done;
        }
        __syncthreads();
        return s_stop != 0;
    };
    // the norm is a by-product of the first pre-smoothing sweep on the finest level
    const bool norm_in_sweep = P.mode == 2 && P.n_pre >= 1;

    for (int cyc = 0;; ++cyc) {
        TP_RESET(cyc, P.mode == 2);
        TP(1);
        if (P.mode == 2 && !norm_in_sweep) {
            if (stop_phase(ph_resnorm<T, D3>(P.g[0], cu[0], P.g[0].rhs, P.a2, w))) break;
            TP(2);
        }
        // (later cycles of a solve loop: the tail's iterate buffers must read as zero again when fewer than two
        // pre-smoothing sweeps overwrite them; ordered before the tail by the barriers of the down leg)
        if (rank == 0 && cyc > 0 && P.n_pre < 2 && P.ntail > 0) tail_zero<T>(P, S);
        // ---- down leg over the cluster levels ----
        bool stop = false;
#pragma unroll 1
        for (int l = 0; l < ng; ++l) {
            const GLevelP<T>& L = P.g[l];
            int s0 = 0;
            if (!(l == 0 && P.mode != 0)) {   // zero initial guess
                if (P.n_pre >= 2) { ph_sweep2_zero<T, D3>(L, L.rhs, cu[l], P.a2, w); s0 = 2; }
                else if (P.n_pre == 1) { ph_scale<T, D3>(L, L.rhs, cu[l], w); s0 = 1; }
                else ph_zero<T, D3>(L, cu[l], w);
                cluster.sync();
                TP(10 * (l + 1) + 0);
            }
            for (int s = s0; s < P.n_pre; ++s) {
                if (l == 0 && s == 0 && norm_in_sweep) {
                    // the sweep goes to the scratch buffer: when the stop rule fires the iterate is still in cu[0]
                    stop = stop_phase(ph_sweep<T, D3, true>(L, cu[l], L.rhs, ct[l], P.a2, w));
                    if (stop) break;
                } else {
                    ph_sweep<T, D3, false>(L, cu[l], L.rhs, ct[l], P.a2, w);
                    cluster.sync();
                }
                T* x = cu[l]; cu[l] = ct[l]; ct[l] = x;
                TP(10 * (l + 1) + 1);
            }
            if (stop) break;
            // the coarse level below: the next cluster level, or the top level of the tail (its global copy)
            const bool last = l + 1 == ng;
            const GLevelP<T>& N = P.g[last ? l : l + 1];
            const int csx = last ? P.tail_sx : N.sx, csy = last ? P.t[0].ny - 1 : N.sy;
            const int cnz = last ? P.t[0].nz : N.nz, csp = last ? P.tail_sp : N.sp;
            T* rc = last ? const_cast<T*>(P.tail_rhs_g) : N.rhs;
            if (!D3) {
                ph_resid_restrict2<T>(L, cu[l], L.rhs, csx, csy, rc, w);
            } else {
                ph_residual<T, D3>(L, cu[l], L.rhs, L.r, P.a2, w);
                cluster.sync();
                TP(10 * (l + 1) + 2);
                ph_restrict<T, D3>(L.r, L.sx, L.sp, csx, csy, cnz, csp, rc, w);
            }
            cluster.sync();
            TP(10 * (l + 1) + 3);
        }
        if (stop) break;
        // ---- tail levels: CTA 0, shared memory ----
        if (rank == 0) tail_body<T, D3>(P, S);
        if (ng > 0) cluster.sync();
        TP(3);
        // ---- up leg ----
#pragma unroll 1
        for (int l = ng - 1; l >= 0; --l) {
            const GLevelP<T>& L = P.g[l];
            const bool last = l + 1 == ng;
            const GLevelP<T>& N = P.g[last ? l : l + 1];
            const T* ec = last ? P.tail_u_g : cu[last ? l : l + 1];
            const int csx = last ? P.tail_sx : N.sx, csp = last ? P.tail_sp : N.sp;
            int s = 0;
            if (!D3 && P.n_post >= 1) {
                ph_prolong_sweep2<T>(L, cu[l], L.rhs, ec, csx, ct[l], w);
                T* x = cu[l]; cu[l] = ct[l]; ct[l] = x;
                s = 1;
            } else {
                ph_prolong<T, D3>(L, cu[l], ec, csx, csp, w);
            }
            cluster.sync();
            TP(10 * (l + 1) + 5);
            for (; s < P.n_post; ++s) {
                ph_sweep<T, D3, false>(L, cu[l], L.rhs, ct[l], P.a2, w);
                T* x = cu[l]; cu[l] = ct[l]; ct[l] = x;
                cluster.sync();
                TP(10 * (l + 1) + 6 + s);
            }
        }
        if (P.mode != 2) break;
    }
    if (P.mode == 2 && rank == 0) {
        __syncthreads();
        const int* src = reinterpret_cast<const int*>(&s_ctl);
        int* dst = reinterpret_cast<int*>(P.ctl);
        for (int q = threadIdx.x; q < (int)(sizeof(Ctl) / sizeof(int)); q += CL_THREADS) dst[q] = src[q];
    }
}

// Which level can start the tail: the first level l >= 1 such that levels l.. fit in `budget` bytes.
int tail_start(const mhs_ctx* c, const std::vector<Level>& Ls, size_t budget)
{
    const int n = (int)Ls.size();
    for (int l = 1; l < n; ++l) {
        if (n - l > 8) continue;  // at most 8 levels in the tail
        size_t bytes = 0;
        for (int q = l; q < n; ++q) bytes += 3 * (size_t)((Ls[q].npts() + 3) & ~3LL) * c->es;
        if (bytes <= budget) return l;
    }
    return n;  // no tail
}

// First level handled by the cluster kernel: the cluster levels [result, tail) are those with at most
// CL_MAX_PTS nodes (and at most CL_MAXG of them); result == tail means "tail only".
int cluster_start(const mhs_ctx* c, const std::vector<Level>& Ls, int tail)
{
    const int n = (int)Ls.size();
    if (tail >= n) return n;   // no tail -> no cluster kernel (the coarsest solve is part of the tail)
    // A hierarchy whose finest level is big keeps only the tail here: its middle levels (<= 129^3) fill the GPU
    // better as ordinary grids (mhs_kernels_fast.cu, mid_level) than on the 16 SMs of one cluster.
    if (Ls[0].dim == 3 && (Ls[0].npts() > CL_MAX_PTS || (c->opt.flags & MHS_FLAG_BIG_LEVEL_KERNELS))) {
        // (tuning knob MHS_CL3_PTS, read at create: levels of a big hierarchy up to that many nodes join the cluster kernel)
        int l = tail;
        while (l > 1 && tail - (l - 1) <= CL_MAXG && Ls[l - 1].npts() <= c->cl3_pts) --l;
        return l;
    }
    int l = tail;
    while (l > 0 && tail - (l - 1) <= CL_MAXG && Ls[l - 1].npts() <= CL_MAX_PTS && Ls[l - 1].sp < (1LL << 30) / std::max(1, Ls[l - 1].nz)) --l;
    return l;
}

// the opt-in dynamic shared memory limit is 227 KB minus the kernel's static shared memory
template <typename K>
static int set_cluster_attrs(K kern)   // returns the limit (bytes of dynamic shared memory)
{
    cudaFuncAttributes fa;
    size_t stat = 4096;
    if (cudaFuncGetAttributes(&fa, kern) == cudaSuccess) stat = fa.sharedSizeBytes;
    const int limit = (int)(227 * 1024 - stat);
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, limit);
    cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaGetLastError();
    return limit;
}

template <typename T, bool D3>
static cudaError_t cluster_launch_t(mhs_ctx* c, std::vector<Level>& Ls, int lc, int mode, const int* done)
{
    ClusterP<T> P;
    memset(&P, 0, sizeof P);
    const int n = (int)Ls.size();
    const int lt = std::max(lc, Ls[0].dim == 3 ? c->tail3 : c->tail2);   // lc > tail: a V pass from inside the tail
    P.mode = mode;
    P.nglob = lt - lc;
    P.ntail = n - lt;
    P.dim3 = D3;
    P.n_pre = c->opt.n_pre; P.n_post = c->opt.n_post;
    P.a2 = D3 ? (T)(c->alpha * c->alpha) : T(0);
    for (int q = lc; q < lt; ++q) {
        const Level& lv = Ls[q];
        GLevelP<T>& g = P.g[q - lc];
        g.nx = lv.nx; g.ny = lv.ny; g.nz = lv.nz; g.sx = lv.sx; g.sy = lv.sy; g.sp = (int)lv.sp;
        g.tab = (const T*)lv.tab;
        g.cz = D3 ? (T)(1.0 / (lv.hz * lv.hz)) : T(0);
        g.u = (T*)lv.u; g.tmp = (T*)lv.tmp; g.rhs = (T*)lv.rhs; g.r = (T*)lv.r;
    }
    int off = 0;
    for (int q = lt; q < n; ++q) {
        const Level& lv = Ls[q];
        TailLevelP<T>& t = P.t[q - lt];
        t.nx = lv.nx; t.ny = lv.ny; t.nz = lv.nz;
        t.bx = 0; while ((1 << t.bx) < lv.nx - 2) ++t.bx;
        t.by = 0; while ((1 << t.by) < lv.ny - 2) ++t.by;
        const int npa = ((int)lv.npts() + 3) & ~3;
        t.off_u = off; t.off_rhs = off + npa; t.off_tmp = off + 2 * npa;
        off += 3 * npa;
        t.tab = (const T*)lv.tab;
        t.cz = D3 ? (T)(1.0 / (lv.hz * lv.hz)) : T(0);
    }
    P.tail_tot = off;
    P.ncoarse = Ls[n - 1].ncoarse;
    P.ainv = (const T*)Ls[n - 1].ainv;
    auto kern = k_cluster<T, D3>;
    static PerDevice dyn_limit;
    const int limit = per_device(dyn_limit, c, [&] { return set_cluster_attrs(kern); });
    // shared copies of the constant data, as far as there is room behind the level arrays: the tables, then the inverse
    for (int q = lt; q < n; ++q) {
        TailLevelP<T>& t = P.t[q - lt];
        const int ne = (4 * Ls[q].nz + 3) & ~3;
        t.off_tab = -1;
        if ((size_t)(off + ne) * sizeof(T) <= (size_t)limit) { t.off_tab = off; off += ne; }
    }
    P.off_ainv = -1;
    if (n > lt) {
        const long long ne = ((long long)P.ncoarse * P.ncoarse + 3) & ~3LL;
        if ((unsigned long long)(off + ne) * sizeof(T) <= (unsigned long long)limit) { P.off_ainv = off; off += (int)ne; }
    }
    P.tail_rhs_g = (const T*)Ls[lt].rhs;
    P.tail_u_g = (T*)Ls[lt].u;
    P.tail_sx = Ls[lt].sx; P.tail_sp = (int)Ls[lt].sp;
    P.partial = c->partial;
    P.ctl = c->ctl;
    const size_t smem = (size_t)off * sizeof(T);

    int ncta = 1;
    if (P.nglob > 0) {
        // enough CTAs that a phase of the largest cluster level is a handful of row segments per warp
        const long long items = Ls[lc].npts() / 32;
        // (measured: the 257^2 solve takes 3.5 / 2.2 / 1.55 / 1.2 ms on 2 / 4 / 8 / 16 CTAs -- phases are chains of L2 round trips,
        // so every halving of the items per thread pays)
        ncta = items > 512 ? c->cluster_max : items > 128 ? std::min(8, c->cluster_max) : items > 32 ? 4 : 2;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ncta);
    cfg.blockDim = dim3(CL_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)ncta; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // PDL, see pdl_enter() in mhs_device.cuh
    at[1].val.programmaticStreamSerializationAllowed = (c->opt.flags & MHS_FLAG_NO_PDL) ? 0 : 1;
    cfg.attrs = at; cfg.numAttrs = 2;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, P, done);
    if (e != cudaSuccess || c->debug)
        fprintf(stderr, "[mhs] k_cluster<%s,%dD> mode %d levels [%d,%d) tail [%d,%d) cluster %d smem %zu: %s\n", sizeof(T) == 8 ? "f64" : "f32",
                D3 ? 3 : 2, mode, lc, lt, lt, n, ncta, smem, cudaGetErrorString(e));
    return e;
}

// Largest cluster (<= 16 CTAs of CL_THREADS threads with the tail's shared memory) this device can co-schedule.
int cluster_max_size(const mhs_ctx* c)
{
    (void)c;
    int best = 1;
    for (int n : {16, 8, 4, 2}) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)n); cfg.blockDim = dim3(CL_THREADS); cfg.dynamicSmemBytes = 216 * 1024;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)n; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        auto kern = k_cluster<double, true>;
        set_cluster_attrs(kern);
        int nc = 0;
        if (cudaOccupancyMaxActiveClusters(&nc, kern, &cfg) == cudaSuccess && nc >= 1) { best = n; break; }
        cudaGetLastError();
    }
    return best;
}

// mode 0: V pass from level lc >= 1 (zero initial guess); mode 1 / 2: lc == 0, one cycle / the whole solve.
// Afterwards Ls[lc].u names the buffer that holds the result when the number of sweeps is known on the host
// (modes 0 and 1); in mode 2 the caller fixes the names up from the cycle count (cluster_fix_names).
void launch_cluster(mhs_ctx* c, std::vector<Level>& Ls, int lc, int mode, const int* done)
{
    count_launch(c);
    cudaError_t e;
    const bool d3 = Ls[0].dim == 3;
    if (c->es == 8) e = d3 ? cluster_launch_t<double, true>(c, Ls, lc, mode, done) : cluster_launch_t<double, false>(c, Ls, lc, mode, done);
    else e = d3 ? cluster_launch_t<float, true>(c, Ls, lc, mode, done) : cluster_launch_t<float, false>(c, Ls, lc, mode, done);
    (void)e;   // surfaced by the caller's cudaGetLastError
    const int lt = d3 ? c->tail3 : c->tail2;
    if (lc < lt && mode != 2) {
        const int np = c->opt.n_pre, nq = c->opt.n_post;
        // (from the zero guess the first two pre-smoothing sweeps are one phase that writes u: no swap)
        const int swaps = (mode == 0 ? (np >= 2 ? np - 2 : 0) : np) + nq;
        if (swaps & 1) std::swap(Ls[lc].u, Ls[lc].tmp);
    }
}

}  // namespace mhs

#ifdef MHS_TAILPROF
// stamps (id, clock64) of the last cycle the cluster kernel recorded; returns their number
extern "C" int mhs_debug_tailprof(long long* out, int cap)
{
    int n = 0;
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(&n, mhs::g_tpn, sizeof n);
    if (n > cap) n = cap;
    cudaMemcpyFromSymbol(out, mhs::g_tp, sizeof(long long) * 2 * n);
    return n;
}
#endif
