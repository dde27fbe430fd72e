// Single-CTA "tail" of the V-cycle: every level small enough to live in one SM's shared memory (u, rhs
// and a scratch array per level, <= ~220 KB in total) is processed by ONE kernel that runs the whole lower
// part of the V -- pre-sweeps, residual, full weighting, the exact coarsest solve, prolongation, post-sweeps
// -- with __syncthreads() between the stages instead of kernel launches.  On those levels the work is a few
// thousand nodes: launch latency, not bandwidth, is what the paper's one-kernel-per-function design
// pays for, and this removes it.  Same arithmetic as the big kernels (mhs_device.cuh).
//
// Shared-memory arrays use the plain dense layout (nx*ny*nz, walls stored as zeros).
#include "mhs_device.cuh"

namespace mhs {

template <typename T>
struct TailLevelP {
    int nx, ny, nz;
    int off_u, off_rhs, off_tmp;  // element offsets into the shared array
    const T* tab;                 // global: cx | cy | diag | w
    T cz;
};

template <typename T>
struct TailP {
    int nlev, dim3, n_pre, n_post, ncoarse;
    T a2;
    TailLevelP<T> lv[8];
    const T* ainv;  // global, ncoarse^2
    const T* rhs_g; // top tail level, aliased layout (in)
    T* u_g;         // top tail level, aliased layout (out)
    int sx;
    long long sp;
};

template <typename T>
__device__ __forceinline__ T tail_Lu(const TailLevelP<T>& L, const T* u, int i, int j, int k, bool d3, T a2)
{
    const int nx = L.nx, nxy = L.nx * L.ny;
    const int c = i + nx * j + nxy * k;
    const T uc = u[c];
    T lu = L.tab[k] * lap1<T>(u[c + 1], u[c - 1], uc) + L.tab[L.nz + k] * lap1<T>(u[c + nx], u[c - nx], uc);
    if (d3) lu += L.cz * lap1<T>(u[c + nxy], u[c - nxy], uc) + a2 * uc;
    return lu;
}

template <typename T>
__global__ void __launch_bounds__(1024) k_tail(TailP<T> P, const int* __restrict__ done)
{
    if (done && *done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* S = reinterpret_cast<T*>(smem_raw);
    const int tid = threadIdx.x, nt = blockDim.x;
    const bool d3 = P.dim3 != 0;

    // zero everything (walls must read as zeros), then load the top level's right-hand side
    int tot = 0;
    {
        const TailLevelP<T>& Ll = P.lv[P.nlev - 1];
        tot = Ll.off_tmp + Ll.nx * Ll.ny * Ll.nz;
        for (int l = 0; l < P.nlev; ++l) {
            const int e = max(max(P.lv[l].off_u, P.lv[l].off_rhs), P.lv[l].off_tmp) + P.lv[l].nx * P.lv[l].ny * P.lv[l].nz;
            tot = max(tot, e);
        }
    }
    for (int q = tid; q < tot; q += nt) S[q] = T(0);
    __syncthreads();
    {
        const TailLevelP<T>& L = P.lv[0];
        const int kz0 = d3 ? 1 : 0, kz1 = d3 ? L.nz - 1 : 1;
        const int mx = L.nx - 2, my = L.ny - 2;
        const int n = mx * my * (kz1 - kz0);
        for (int q = tid; q < n; q += nt) {
            const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
            S[L.off_rhs + i + L.nx * j + L.nx * L.ny * k] = P.rhs_g[i + (long long)P.sx * j + P.sp * k];
        }
    }
    __syncthreads();

    // ---- down leg ----
    for (int l = 0; l < P.nlev - 1; ++l) {
        const TailLevelP<T>& L = P.lv[l];
        const TailLevelP<T>& C = P.lv[l + 1];
        const int kz0 = d3 ? 1 : 0, kz1 = d3 ? L.nz - 1 : 1;
        const int mx = L.nx - 2, my = L.ny - 2, n = mx * my * (kz1 - kz0);
        T* u = S + L.off_u;
        T* tmp = S + L.off_tmp;
        const T* rhs = S + L.off_rhs;
        // u starts from zero (it was cleared above / by the previous use): sweeps
        for (int q = tid; q < L.nx * L.ny * L.nz; q += nt) u[q] = T(0);
        __syncthreads();
        for (int s = 0; s < P.n_pre; ++s) {
            for (int q = tid; q < n; q += nt) {
                const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
                const int c = i + L.nx * j + L.nx * L.ny * k;
                tmp[c] = u[c] + L.tab[3 * L.nz + k] * (rhs[c] - tail_Lu<T>(L, u, i, j, k, d3, P.a2));
            }
            __syncthreads();
            for (int q = tid; q < n; q += nt) {
                const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
                const int c = i + L.nx * j + L.nx * L.ny * k;
                u[c] = tmp[c];
            }
            __syncthreads();
        }
        // residual -> tmp
        for (int q = tid; q < n; q += nt) {
            const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
            const int c = i + L.nx * j + L.nx * L.ny * k;
            tmp[c] = rhs[c] - tail_Lu<T>(L, u, i, j, k, d3, P.a2);
        }
        __syncthreads();
        // full weighting -> rhs of the next level
        {
            const int cmx = C.nx - 2, cmy = C.ny - 2;
            const int ck0 = d3 ? 1 : 0, ck1 = d3 ? C.nz - 1 : 1;
            const int cn = cmx * cmy * (ck1 - ck0);
            T* rc = S + C.off_rhs;
            for (int q = tid; q < cn; q += nt) {
                const int I = q % cmx + 1, J = (q / cmx) % cmy + 1, K = q / (cmx * cmy) + ck0;
                const T* r0 = tmp + 2 * I + L.nx * (2 * J) + L.nx * L.ny * (2 * K);
                T s = T(0);
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
                rc[I + C.nx * J + C.nx * C.ny * K] = s;
            }
        }
        __syncthreads();
    }

    // ---- coarsest level: exact solve e = A^-1 rhs ----
    {
        const TailLevelP<T>& L = P.lv[P.nlev - 1];
        const int mx = L.nx - 2, my = L.ny - 2, k0 = d3 ? 1 : 0;
        const int n = P.ncoarse;
        T* u = S + L.off_u;
        const T* rhs = S + L.off_rhs;
        for (int row = tid; row < n; row += nt) {
            double s = 0.0;
            for (int col = 0; col < n; ++col) {
                const int ci = col % mx, cj = (col / mx) % my, ck = col / (mx * my);
                s += (double)P.ainv[(long long)row * n + col] * (double)rhs[(ci + 1) + L.nx * (cj + 1) + L.nx * L.ny * (ck + k0)];
            }
            const int i = row % mx, j = (row / mx) % my, k = row / (mx * my);
            u[(i + 1) + L.nx * (j + 1) + L.nx * L.ny * (k + k0)] = (T)s;
        }
        __syncthreads();
    }

    // ---- up leg ----
    for (int l = P.nlev - 2; l >= 0; --l) {
        const TailLevelP<T>& L = P.lv[l];
        const TailLevelP<T>& C = P.lv[l + 1];
        const int kz0 = d3 ? 1 : 0, kz1 = d3 ? L.nz - 1 : 1;
        const int mx = L.nx - 2, my = L.ny - 2, n = mx * my * (kz1 - kz0);
        T* u = S + L.off_u;
        T* tmp = S + L.off_tmp;
        const T* rhs = S + L.off_rhs;
        const T* ec = S + C.off_u;
        for (int q = tid; q < n; q += nt) {
            const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
            const int I0 = i >> 1, I1 = (i + 1) >> 1, J0 = j >> 1, J1 = (j + 1) >> 1, K0 = k >> 1, K1 = (k + 1) >> 1;
            const int cxy = C.nx * C.ny;
            T s = (ec[I0 + C.nx * J0 + cxy * K0] + ec[I1 + C.nx * J0 + cxy * K0]) +
                  (ec[I0 + C.nx * J1 + cxy * K0] + ec[I1 + C.nx * J1 + cxy * K0]);
            if (d3)
                s += (ec[I0 + C.nx * J0 + cxy * K1] + ec[I1 + C.nx * J0 + cxy * K1]) +
                     (ec[I0 + C.nx * J1 + cxy * K1] + ec[I1 + C.nx * J1 + cxy * K1]);
            u[i + L.nx * j + L.nx * L.ny * k] += (d3 ? T(0.125) : T(0.25)) * s;
        }
        __syncthreads();
        for (int s = 0; s < P.n_post; ++s) {
            for (int q = tid; q < n; q += nt) {
                const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
                const int c = i + L.nx * j + L.nx * L.ny * k;
                tmp[c] = u[c] + L.tab[3 * L.nz + k] * (rhs[c] - tail_Lu<T>(L, u, i, j, k, d3, P.a2));
            }
            __syncthreads();
            for (int q = tid; q < n; q += nt) {
                const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
                const int c = i + L.nx * j + L.nx * L.ny * k;
                u[c] = tmp[c];
            }
            __syncthreads();
        }
    }

    // ---- write the correction of the top tail level back (interior nodes) ----
    {
        const TailLevelP<T>& L = P.lv[0];
        const int kz0 = d3 ? 1 : 0, kz1 = d3 ? L.nz - 1 : 1;
        const int mx = L.nx - 2, my = L.ny - 2, n = mx * my * (kz1 - kz0);
        const T* u = S + L.off_u;
        for (int q = tid; q < n; q += nt) {
            const int i = q % mx + 1, j = (q / mx) % my + 1, k = q / (mx * my) + kz0;
            P.u_g[i + (long long)P.sx * j + P.sp * k] = u[i + L.nx * j + L.nx * L.ny * k];
        }
    }
}

// Which level can start the tail: the first level l >= 1 such that levels l.. fit in `budget` bytes.
int tail_start(const mhs_ctx* c, const std::vector<Level>& Ls, size_t budget)
{
    const int n = (int)Ls.size();
    if (n - 1 > 8) {
        // at most 8 levels in the tail
    }
    for (int l = 1; l < n; ++l) {
        if (n - l > 8) continue;
        size_t bytes = 0;
        for (int q = l; q < n; ++q) bytes += 3 * (size_t)Ls[q].npts() * c->es;
        if (bytes <= budget) return l;
    }
    return n;  // no tail
}

template <typename T>
static void tail_t(mhs_ctx* c, std::vector<Level>& Ls, int l0, const int* done)
{
    TailP<T> P;
    memset(&P, 0, sizeof P);
    const int n = (int)Ls.size();
    P.nlev = n - l0;
    P.dim3 = Ls[l0].dim == 3;
    P.n_pre = c->opt.n_pre; P.n_post = c->opt.n_post;
    P.a2 = P.dim3 ? (T)(c->alpha * c->alpha) : T(0);
    int off = 0;
    for (int q = l0; q < n; ++q) {
        const Level& lv = Ls[q];
        TailLevelP<T>& t = P.lv[q - l0];
        t.nx = lv.nx; t.ny = lv.ny; t.nz = lv.nz;
        const int np = (int)lv.npts();
        const int npa = (np + 3) & ~3;
        t.off_u = off; t.off_rhs = off + npa; t.off_tmp = off + 2 * npa;
        off += 3 * npa;
        t.tab = (const T*)lv.tab;
        t.cz = P.dim3 ? (T)(1.0 / (lv.hz * lv.hz)) : T(0);
    }
    P.ncoarse = Ls[n - 1].ncoarse;
    P.ainv = (const T*)Ls[n - 1].ainv;
    P.rhs_g = (const T*)Ls[l0].rhs;
    P.u_g = (T*)Ls[l0].u;
    P.sx = Ls[l0].sx; P.sp = Ls[l0].sp;
    const size_t smem = (size_t)off * sizeof(T);
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_tail<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        attr_set = true;
    }
    k_tail<T><<<1, 1024, smem, c->stream>>>(P, done);
}

void launch_tail(mhs_ctx* c, std::vector<Level>& Ls, int l0, const int* done)
{
    count_launch(c);
    if (c->es == 8) tail_t<double>(c, Ls, l0, done);
    else tail_t<float>(c, Ls, l0, done);
}

}  // namespace mhs
