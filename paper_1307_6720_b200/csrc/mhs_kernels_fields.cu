// Field recovery of libmhs_b200 for sm_100a (a8 + a9; eqs 9-10; readings C13-C15):
//   Bz = -(dxx + dyy) P,  Bx = alpha D_y P + D_x D_z P,  By = -alpha D_x P + D_y D_z P,
//   p = p_b - xi Bz^2/(2 mu0),  rho = rho_b + (1/g) [ xi' Bz^2/(2 mu0) + (xi/mu0) B . grad Bz ]
// ONE pass: P is read once from HBM and the five outputs are written once (6w bytes per node) -- Bz, which the
// density needs at all six neighbours, is never read back: a thread owns one 128-bit vector of one row and walks
// up in z carrying the planes k-1, k, k+1 of P AND of Bz for its nodes in registers; x-neighbours come from warp
// shuffles (the flat aliased layout makes the neighbour across a row end the wall zero), y-neighbours from the
// rows of the other warps of the block through the L1.  Outputs are DENSE (pitch nx, the ABI layout), so the
// aliased wall nodes (nx-1, j) and the row ny-1 are written by the threads that own their aliases.
// The planes k = 0 (one-sided z differences, C13) and k = nz-1 (all wall) are left to the reference kernel.
#include "mhs_device.cuh"

namespace mhs {

template <typename T> struct FV;
template <> struct FV<double> { static constexpr int N = 2; };
template <> struct FV<float> { static constexpr int N = 4; };

template <typename T>
struct __align__(16) FVec {
    T v[FV<T>::N];
};
template <typename T>
__device__ __forceinline__ FVec<T> fld(const T* p) { return *reinterpret_cast<const FVec<T>*>(p); }

template <typename T>
struct FZP {
    int nx, ny, nz, sx, sy;
    long long sp;
    T alpha, i2hx, i2hy, i2hz, ihx2, ihy2, i2mu0, imu0, ig;
    const T* ft;   // xi[nz] | dxi[nz] | p_b[nz] | rho_b[nz]
};

__device__ __forceinline__ double f_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float f_up(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double f_dn(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float f_dn(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// left / right x-neighbours of every element of a vector: inside the vector, else the neighbouring lane's edge
// element, else (lanes 0 / 31) the separately loaded values wl / wr.
template <typename T>
__device__ __forceinline__ void xnb(const FVec<T>& c, T wl, T wr, int lane, T* L, T* R)
{
    constexpr int V = FV<T>::N;
    T l = f_up(c.v[V - 1]), r = f_dn(c.v[0]);
    if (lane == 0) l = wl;
    if (lane == 31) r = wr;
#pragma unroll
    for (int e = 0; e < V; ++e) {
        L[e] = e == 0 ? l : c.v[e - 1];
        R[e] = e == V - 1 ? r : c.v[e + 1];
    }
}

// -(dxx + dyy) of one vector, same arithmetic as the reference kernel's Bz_at
template <typename T>
__device__ __forceinline__ void bz_vec(const FZP<T>& q, const FVec<T>& c, const T* L, const T* R, const FVec<T>& n, const FVec<T>& s, T* bz)
{
#pragma unroll
    for (int e = 0; e < FV<T>::N; ++e) {
        const T dxx = (R[e] - T(2) * c.v[e] + L[e]) * q.ihx2;
        const T dyy = (n.v[e] - T(2) * c.v[e] + s.v[e]) * q.ihy2;
        bz[e] = -(dxx + dyy);
    }
}

// block (32, 8): warp y owns row j0 + y, lane x the vector i0 = (blockIdx.x*32 + x)*V of that row.
template <typename T>
__global__ void __launch_bounds__(256) k_fields_z(const FZP<T> q, const T* __restrict__ P, T* __restrict__ Bx, T* __restrict__ By,
                                                   T* __restrict__ Bzo, T* __restrict__ pp, T* __restrict__ rho, int kchunk)
{
    constexpr int V = FV<T>::N;
    const int lane = threadIdx.x;
    const int i0 = (blockIdx.x * 32 + lane) * V;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (j >= q.sy) return;                        // whole warps only (blockDim.y rows per block)
    const int kb = 1 + blockIdx.z * kchunk;
    const int ke = min(kb + kchunk, q.nz - 1);    // output planes [kb, ke), all interior in z
    if (kb >= ke) return;
    const int sx = q.sx;
    const long long sp = q.sp;
    const T* base = P + i0 + (long long)sx * j;   // own vector, plane 0
    const bool edge = lane == 0 || lane == 31;
    const int side = lane == 0 ? -1 : V;          // column offset of the neighbour an edge lane has to fetch itself
    const int side2 = lane == 0 ? -2 : V + 1;
    // wall masks.  Nodes i = nx-1 and j = ny-1 do not exist in the aliased layout (they are (0, j+1) and row 0).
    const bool row_wall = j == 0;
    const bool n_wall = j + 1 >= q.sy, s_wall = j - 1 <= 0;   // rows j+1 / j-1 are wall rows
    bool ewall[V];
#pragma unroll
    for (int e = 0; e < V; ++e) ewall[e] = row_wall || (i0 + e == 0);
    const bool side_wall = row_wall || (i0 + side <= 0) || (i0 + side >= sx);   // the edge lane's neighbour node is a wall

    // Bz of this thread's vector on plane k (0 at wall nodes), given the plane's centre, north and south vectors
    auto own_bz = [&](const T* pl, const FVec<T>& c, const FVec<T>& n, const FVec<T>& s, bool top, T* bz) {
        T wl = T(0), wr = T(0);
        if (edge) { const T w = pl[side]; if (lane == 0) wl = w; else wr = w; }
        T L[V], R[V];
        xnb<T>(c, wl, wr, lane, L, R);
        bz_vec<T>(q, c, L, R, n, s, bz);
#pragma unroll
        for (int e = 0; e < V; ++e)
            if (ewall[e] || top) bz[e] = T(0);
    };

    FVec<T> Pm = fld(base + sp * (kb - 1)), Pc = fld(base + sp * kb);
    T bzm[V], bzc[V];
    {
        const T* pm = base + sp * (kb - 1);
        own_bz(pm, Pm, fld(pm + sx), fld(pm - sx), false, bzm);
        const T* pc = base + sp * kb;
        own_bz(pc, Pc, fld(pc + sx), fld(pc - sx), false, bzc);
    }

    for (int k = kb; k < ke; ++k) {
        const T* pc = base + sp * k;
        const T* pu = pc + sp;
        const T* pd = pc - sp;
        const FVec<T> Pp = fld(pu);
        const FVec<T> Pn_p = fld(pu + sx), Ps_p = fld(pu - sx);
        const FVec<T> Pn_m = fld(pd + sx), Ps_m = fld(pd - sx);
        const FVec<T> Pn_c = fld(pc + sx), Ps_c = fld(pc - sx);
        const FVec<T> Pnn = fld(pc + 2 * sx), Pss = fld(pc - 2 * sx);
        const T xi = q.ft[k], dxi = q.ft[q.nz + k], pb = q.ft[2 * q.nz + k], rb = q.ft[3 * q.nz + k];

        // Bz of the own nodes on plane k+1 (the top plane is a wall)
        T bzp[V];
        own_bz(pu, Pp, Pn_p, Ps_p, k + 1 >= q.nz - 1, bzp);

        // what the edge lanes fetch for the neighbour column i0 + side of row j
        T ePc = T(0), edz = T(0), ebz = T(0), ePn = T(0), ePs = T(0);
        if (edge) {
            ePc = pc[side];
            edz = (pu[side] - pd[side]) * q.i2hz;
            ePn = pc[sx + side];
            ePs = pc[side - sx];
            const T far = pc[side2];
            const T near = lane == 0 ? Pc.v[0] : Pc.v[V - 1];
            const T dxx = ((lane == 0 ? near : far) - T(2) * ePc + (lane == 0 ? far : near)) * q.ihx2;
            const T dyy = (ePn - T(2) * ePc + ePs) * q.ihy2;
            ebz = side_wall ? T(0) : -(dxx + dyy);
        }
        // x-neighbours of P, D_z P and Bz on plane k
        FVec<T> dz, bzv;
#pragma unroll
        for (int e = 0; e < V; ++e) { dz.v[e] = (Pp.v[e] - Pm.v[e]) * q.i2hz; bzv.v[e] = bzc[e]; }
        T PL[V], PR[V], dzL[V], dzR[V], bL[V], bR[V], nL[V], nR[V], sL[V], sR[V];
        xnb<T>(Pc, ePc, ePc, lane, PL, PR);
        xnb<T>(dz, edz, edz, lane, dzL, dzR);
        xnb<T>(bzv, ebz, ebz, lane, bL, bR);
        xnb<T>(Pn_c, ePn, ePn, lane, nL, nR);
        xnb<T>(Ps_c, ePs, ePs, lane, sL, sR);
        // Bz on the rows j+1 / j-1 of plane k (0 on wall rows and wall columns)
        T bzn[V], bzs[V];
        bz_vec<T>(q, Pn_c, nL, nR, Pnn, Pc, bzn);
        bz_vec<T>(q, Ps_c, sL, sR, Pc, Pss, bzs);
#pragma unroll
        for (int e = 0; e < V; ++e) {
            if (n_wall || i0 + e == 0) bzn[e] = T(0);
            if (s_wall || i0 + e == 0) bzs[e] = T(0);
        }

        const long long drow = (long long)q.nx * (j + (long long)q.ny * k);
#pragma unroll
        for (int e = 0; e < V; ++e) {
            T bx = T(0), by = T(0), bz = T(0), pv = pb, rv = rb;
            if (!ewall[e]) {
                bz = bzc[e];
                const T dzn = (Pn_p.v[e] - Pn_m.v[e]) * q.i2hz, dzs = (Ps_p.v[e] - Ps_m.v[e]) * q.i2hz;
                bx = q.alpha * (Pn_c.v[e] - Ps_c.v[e]) * q.i2hy + (dzR[e] - dzL[e]) * q.i2hx;
                by = -q.alpha * (PR[e] - PL[e]) * q.i2hx + (dzn - dzs) * q.i2hy;
                const T dxBz = (bR[e] - bL[e]) * q.i2hx;
                const T dyBz = (bzn[e] - bzs[e]) * q.i2hy;
                const T dzBz = (bzp[e] - bzm[e]) * q.i2hz;
                pv = pb - xi * bz * bz * q.i2mu0;
                rv = rb + q.ig * (dxi * bz * bz * q.i2mu0 + q.imu0 * xi * (bx * dxBz + by * dyBz + bz * dzBz));
            }
            const long long d = drow + i0 + e;
            if (Bx) { Bx[d] = bx; By[d] = by; Bzo[d] = bz; }
            if (pp) pp[d] = pv;
            if (rho) rho[d] = rv;
        }
        // the aliased wall nodes: (nx-1, j) belongs to the thread that owns (0, j); row ny-1 to the warps of row 0
        if (i0 == 0) {
            const long long d = drow + q.nx - 1;
            if (Bx) { Bx[d] = T(0); By[d] = T(0); Bzo[d] = T(0); }
            if (pp) pp[d] = pb;
            if (rho) rho[d] = rb;
        }
        if (row_wall) {
            const long long dtop = (long long)q.nx * (q.ny - 1 + (long long)q.ny * k);
#pragma unroll
            for (int e = 0; e < V; ++e) {
                const long long d = dtop + i0 + e;
                if (Bx) { Bx[d] = T(0); By[d] = T(0); Bzo[d] = T(0); }
                if (pp) pp[d] = pb;
                if (rho) rho[d] = rb;
            }
            if (i0 == 0) {
                const long long d = dtop + q.nx - 1;
                if (Bx) { Bx[d] = T(0); By[d] = T(0); Bzo[d] = T(0); }
                if (pp) pp[d] = pb;
                if (rho) rho[d] = rb;
            }
        }
        Pm = Pc; Pc = Pp;
#pragma unroll
        for (int e = 0; e < V; ++e) { bzm[e] = bzc[e]; bzc[e] = bzp[e]; }
    }
}

bool fields_z_ok(const mhs_ctx* c, const Level& lv)
{
    const int V = c->es == 8 ? 2 : 4;
    return lv.dim == 3 && lv.sx % (32 * V) == 0 && lv.sy % 8 == 0 && lv.nz >= 5;
}

template <typename T>
static void fields_z_t(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho)
{
    constexpr int V = FV<T>::N;
    FZP<T> q;
    q.nx = lv.nx; q.ny = lv.ny; q.nz = lv.nz; q.sx = lv.sx; q.sy = lv.sy; q.sp = lv.sp;
    q.alpha = (T)c->alpha;
    q.i2hx = (T)(1.0 / (2.0 * lv.hx)); q.i2hy = (T)(1.0 / (2.0 * lv.hy)); q.i2hz = (T)(1.0 / (2.0 * lv.hz));
    q.ihx2 = (T)(1.0 / (lv.hx * lv.hx)); q.ihy2 = (T)(1.0 / (lv.hy * lv.hy));
    q.i2mu0 = (T)(1.0 / (2.0 * c->opt.mu0)); q.imu0 = (T)(1.0 / c->opt.mu0); q.ig = (T)(1.0 / c->opt.g);
    q.ft = (const T*)c->prof_tab;
    auto kern = k_fields_z<T>;
    static PerDevice slots_pd;
    const int slots = per_device(slots_pd, c, [&] {
        prefer_l1(kern);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 256, 0);
        return std::max(1, nb) * c->num_sms;
    });
    const int bx = lv.sx / (32 * V), by = lv.sy / 8;
    const int planes = lv.nz - 2;
    // z-chunks: about two waves of blocks, chunks no shorter than 8 planes (2 warm-up planes each)
    int nzc = std::max(1, std::min(planes / 8, (2 * slots + bx * by - 1) / (bx * by)));
    const int kchunk = (planes + nzc - 1) / nzc;
    nzc = (planes + kchunk - 1) / kchunk;
    const long long N = lv.npts();
    T* Bp = (T*)B;
    kern<<<dim3(bx, by, nzc), dim3(32, 8), 0, c->stream>>>(q, (const T*)P, Bp, Bp ? Bp + N : nullptr, Bp ? Bp + 2 * N : nullptr, (T*)p,
                                                         (T*)rho, kchunk);
}

// planes 1 .. nz-2 of B, p, rho (the caller gives planes 0 and nz-1 to the reference kernel)
void launch_fields_z(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho)
{
    count_launch(c);
    if (c->es == 8) fields_z_t<double>(c, lv, P, B, p, rho);
    else fields_z_t<float>(c, lv, P, B, p, rho);
}

// ------------------------------------------------------------------------------------------------
// Diagnostics (the quantities of the paper's Figs 2, 4-7): |B| and j = curl B / mu0 (eq 2,
// PAPER.md:41) with |j|, from the dense B that mhs_fields returns.  Second-order central differences, one-sided second
// order in z on the bottom plane (as for B itself, C13); j = 0 on the side and top boundary nodes, where B = 0 is imposed
// (PAPER.md:134).  One thread per node: 3w read + up to 5w written per node, dense in and out.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_diagnostics(int nx, int ny, int nz, T i2hx, T i2hy, T i2hz, T imu0, const T* __restrict__ Bx,
                                                      const T* __restrict__ By, const T* __restrict__ Bz, T* __restrict__ absB,
                                                      T* __restrict__ Jx, T* __restrict__ Jy, T* __restrict__ Jz, T* __restrict__ absJ)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= nx || j >= ny) return;
    const long long sy = nx, sz = (long long)nx * ny;
    const long long q = i + sy * j + sz * k;
    const T bx = Bx[q], by = By[q], bz = Bz[q];
    if (absB) absB[q] = sqrt(bx * bx + by * by + bz * bz);
    T a = T(0), b = T(0), c = T(0);
    const bool wall = i == 0 || i == nx - 1 || j == 0 || j == ny - 1 || k == nz - 1;
    if (!wall) {
        const T dyBz = (Bz[q + sy] - Bz[q - sy]) * i2hy, dxBz = (Bz[q + 1] - Bz[q - 1]) * i2hx;
        const T dxBy = (By[q + 1] - By[q - 1]) * i2hx, dyBx = (Bx[q + sy] - Bx[q - sy]) * i2hy;
        T dzBy, dzBx;
        if (k == 0) {
            dzBy = (T(-3) * by + T(4) * By[q + sz] - By[q + 2 * sz]) * i2hz;
            dzBx = (T(-3) * bx + T(4) * Bx[q + sz] - Bx[q + 2 * sz]) * i2hz;
        } else {
            dzBy = (By[q + sz] - By[q - sz]) * i2hz;
            dzBx = (Bx[q + sz] - Bx[q - sz]) * i2hz;
        }
        a = (dyBz - dzBy) * imu0; b = (dzBx - dxBz) * imu0; c = (dxBy - dyBx) * imu0;
    }
    if (Jx) { Jx[q] = a; Jy[q] = b; Jz[q] = c; }
    if (absJ) absJ[q] = sqrt(a * a + b * b + c * c);
}

template <typename T>
static void diagnostics_t(mhs_ctx* c, const Level& lv, const void* B, void* absB, void* J, void* absJ)
{
    static PerDevice once;
    per_device(once, c, [&] { prefer_l1(k_diagnostics<T>); return 1; });
    const long long N = lv.npts();
    const T* Bp = (const T*)B;
    T* Jp = (T*)J;
    const dim3 b(32, 8), g((lv.nx + 31) / 32, (lv.ny + 7) / 8, lv.nz);
    k_diagnostics<T><<<g, b, 0, c->stream>>>(lv.nx, lv.ny, lv.nz, (T)(1.0 / (2.0 * lv.hx)), (T)(1.0 / (2.0 * lv.hy)), (T)(1.0 / (2.0 * lv.hz)),
                                             (T)(1.0 / c->opt.mu0), Bp, Bp + N, Bp + 2 * N, (T*)absB, Jp, Jp ? Jp + N : nullptr,
                                             Jp ? Jp + 2 * N : nullptr, (T*)absJ);
}

void launch_diagnostics(mhs_ctx* c, const Level& lv, const void* B, void* absB, void* J, void* absJ)
{
    count_launch(c);
    if (c->es == 8) diagnostics_t<double>(c, lv, B, absB, J, absJ);
    else diagnostics_t<float>(c, lv, B, absB, J, absJ);
}

}  // namespace mhs
