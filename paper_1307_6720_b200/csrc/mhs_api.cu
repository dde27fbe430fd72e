// C ABI of libmhs_b200 (include/mhs.h): context + level hierarchy, V-cycle driver, solve loops.
// Host logic only -- every arithmetic step of the path runs in the kernels of mhs_kernels_*.cu.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "mhs_device.cuh"

using namespace mhs;

namespace {

#define CK(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            ctx->err = std::string(#call) + ": " + cudaGetErrorString(e_);                               \
            return e_ == cudaErrorMemoryAllocation ? MHS_ERR_OOM : MHS_ERR_CUDA;                         \
        }                                                                                                \
    } while (0)

// The control block goes back to the host by STORES into mapped pinned memory, not by a DMA copy: a copy would queue on
// the device->host copy engine behind the 679 MB of field results that mhs_fields_host_async may have in flight, and the
// solve loop of the next step would stall on it.
__global__ void k_ctl_to_host(const Ctl* __restrict__ ctl, Ctl* host)
{
    pdl_enter();
    const int n = (int)(sizeof(Ctl) / sizeof(int));
    const int* s = reinterpret_cast<const int*>(ctl);
    int* d = reinterpret_cast<int*>(host);
    for (int i = threadIdx.x; i < n; i += blockDim.x) d[i] = s[i];
    __threadfence_system();
}

mhs_status read_ctl(mhs_ctx* ctx)
{
    launch_pdl(ctx, k_ctl_to_host, dim3(1), dim3(256), 0, (const Ctl*)ctx->ctl, ctx->ctl_host);
    cudaError_t e_ = cudaStreamSynchronize(ctx->stream);
    if (e_ != cudaSuccess) {
        ctx->err = std::string("cudaStreamSynchronize: ") + cudaGetErrorString(e_);
        return MHS_ERR_CUDA;
    }
    return MHS_OK;
}

mhs_status fail(mhs_ctx* ctx, mhs_status s, const std::string& msg)
{
    ctx->err = msg;
    return s;
}

// RAII kernel-class scope: routes launch counts, and CUDA-event timing when profiling is on.
struct Scope {
    mhs_ctx* c;
    int prev;
    bool timed;
    Ev ev{};
    Scope(mhs_ctx* ctx, int kc) : c(ctx), prev(ctx->cur_kc)
    {
        c->cur_kc = kc;
        timed = c->opt.profile >= 2 || (c->opt.profile == 1 && (kc == MHS_KC_SMOOTH_L0 || kc == MHS_KC_PROLONG_L0));
        if (timed) {
            ev.kc = kc;
            ev.a = take();
            ev.b = take();
            cudaEventRecord(ev.a, c->stream);
        }
    }
    ~Scope()
    {
        if (timed) {
            cudaEventRecord(ev.b, c->stream);
            c->ev_pending.push_back(ev);
        }
        c->cur_kc = prev;
    }
    cudaEvent_t take()
    {
        if (!c->ev_pool.empty()) {
            cudaEvent_t e = c->ev_pool.back();
            c->ev_pool.pop_back();
            return e;
        }
        cudaEvent_t e;
        cudaEventCreate(&e);
        return e;
    }
};

// After a stream synchronisation: fold finished event pairs into the profile.
void drain_events(mhs_ctx* c)
{
    for (const Ev& e : c->ev_pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) c->prof.ms[e.kc] += ms;
        c->ev_pool.push_back(e.a);
        c->ev_pool.push_back(e.b);
    }
    c->ev_pending.clear();
}

// Dense inverse by Gauss-Jordan with partial pivoting (fp64, host).  A is n x n row-major, overwritten by A^-1.
bool invert_dense(int n, std::vector<double>& A)
{
    std::vector<double> M((size_t)n * 2 * n, 0.0);
    for (int r = 0; r < n; ++r) {
        for (int c = 0; c < n; ++c) M[(size_t)r * 2 * n + c] = A[(size_t)r * n + c];
        M[(size_t)r * 2 * n + n + r] = 1.0;
    }
    for (int col = 0; col < n; ++col) {
        int piv = col;
        double best = std::fabs(M[(size_t)col * 2 * n + col]);
        for (int r = col + 1; r < n; ++r) {
            double v = std::fabs(M[(size_t)r * 2 * n + col]);
            if (v > best) { best = v; piv = r; }
        }
        if (best == 0.0) return false;
        if (piv != col)
            for (int c = 0; c < 2 * n; ++c) std::swap(M[(size_t)col * 2 * n + c], M[(size_t)piv * 2 * n + c]);
        const double d = 1.0 / M[(size_t)col * 2 * n + col];
        for (int c = 0; c < 2 * n; ++c) M[(size_t)col * 2 * n + c] *= d;
        for (int r = 0; r < n; ++r) {
            if (r == col) continue;
            const double m = M[(size_t)r * 2 * n + col];
            if (m == 0.0) continue;
            for (int c = 0; c < 2 * n; ++c) M[(size_t)r * 2 * n + c] -= m * M[(size_t)col * 2 * n + c];
        }
    }
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) A[(size_t)r * n + c] = M[(size_t)r * 2 * n + n + c];
    return true;
}

bool level_is_coarsest(int nx, int ny, int nz, int dim, int level, int max_levels)
{
    if (max_levels > 0 && level + 1 >= max_levels) return true;
    const int mx = nx - 1, my = ny - 1, mz = nz - 1;
    if ((mx & 1) || mx < 4 || (my & 1) || my < 4) return true;
    if (dim == 3 && ((mz & 1) || mz < 4)) return true;
    return false;
}

template <typename T>
std::vector<T> cast_vec(const std::vector<double>& v)
{
    std::vector<T> o(v.size());
    for (size_t i = 0; i < v.size(); ++i) o[i] = (T)v[i];
    return o;
}

mhs_status upload(mhs_ctx* ctx, void** dst, const std::vector<double>& v)
{
    CK(cudaMalloc(dst, v.size() * ctx->es));
    if (ctx->es == 8) {
        CK(cudaMemcpy(*dst, v.data(), v.size() * 8, cudaMemcpyHostToDevice));
    } else {
        std::vector<float> f = cast_vec<float>(v);
        CK(cudaMemcpy(*dst, f.data(), f.size() * 4, cudaMemcpyHostToDevice));
    }
    return MHS_OK;
}

mhs_status alloc_field(mhs_ctx* ctx, Level& lv, int slot, void** out)
{
    void* raw = nullptr;
    CK(cudaMalloc(&raw, (size_t)lv.alloc * ctx->es));
    CK(cudaMemset(raw, 0, (size_t)lv.alloc * ctx->es));
    lv.raw[slot] = raw;
    *out = (char*)raw + (size_t)lv.pad * ctx->es;
    return MHS_OK;
}

// Build one hierarchy (dim 2 or 3): extents, spacings, coefficient tables, coarsest inverse, arrays.
mhs_status build_hierarchy(mhs_ctx* ctx, int dim, std::vector<Level>& Ls)
{
    const mhs_grid& g = ctx->grid;
    int nx = g.nx, ny = g.ny, nz = dim == 3 ? g.nz : 1;
    double hx = g.Lx / (g.nx - 1), hy = g.Ly / (g.ny - 1), hz = dim == 3 ? g.Lz / (g.nz - 1) : 0.0;
    std::vector<double> c(nz, 1.0);
    if (dim == 3)
        for (int k = 0; k < nz; ++k) c[k] = 1.0 + ctx->f[k];
    const double a2 = dim == 3 ? ctx->alpha * ctx->alpha : 0.0;
    for (int l = 0;; ++l) {
        Level lv;
        lv.dim = dim; lv.nx = nx; lv.ny = ny; lv.nz = nz; lv.sx = nx - 1; lv.sy = ny - 1;
        lv.sp = (long long)lv.sx * lv.sy;
        lv.hx = hx; lv.hy = hy; lv.hz = hz; lv.c = c;
        lv.coarsest = level_is_coarsest(nx, ny, nz, dim, l, ctx->opt.max_levels);
        const long long front = (dim == 3 ? lv.sp : 0) + lv.sx + 32;
        lv.pad = (front + 31) / 32 * 32;
        lv.alloc = lv.pad + lv.sp * nz + (dim == 3 ? lv.sp : 0) + lv.sx + 64;
        // coefficient table: cx | cy | diag | w | A | Bx | By | Bz | iw | wz.  The last six are the per-plane
        // coefficients of the expanded Jacobi update u' = A u + Bx (e+w) + By (n+s) + Bz (up+dn) + wz f used by
        // the temporally blocked smoother (mhs_kernels_zfused.cu): A = 1-omega, Bx = -w cx, ..., iw = 1/w = D/omega;
        // on the fixed planes k = 0 and k = nz-1 of a 3D level they read A = 1, B = 0, wz = 0: "copy through".
        std::vector<double> tab(10 * (size_t)nz);
        for (int k = 0; k < nz; ++k) {
            const double cx = c[k] / (hx * hx), cy = c[k] / (hy * hy);
            const double d = -2.0 * cx - 2.0 * cy - (dim == 3 ? 2.0 / (hz * hz) : 0.0) + a2;
            const bool interior = dim == 2 || (k > 0 && k < nz - 1);
            if (interior && !(d < 0.0)) {
                char b[160];
                snprintf(b, sizeof b, "operator not negative definite: diagonal D_k = %g >= 0 on level %d, plane %d (alpha^2 too large)", d, l, k);
                return fail(ctx, MHS_ERR_INDEFINITE, b);
            }
            tab[k] = cx; tab[nz + k] = cy; tab[2 * nz + k] = d; tab[3 * nz + k] = ctx->opt.omega / d;
            const double w = ctx->opt.omega / d;
            const size_t n = (size_t)nz;
            if (interior) {
                tab[4 * n + k] = 1.0 - ctx->opt.omega; tab[5 * n + k] = -w * cx; tab[6 * n + k] = -w * cy;
                tab[7 * n + k] = dim == 3 ? -w / (hz * hz) : 0.0; tab[8 * n + k] = 1.0 / w; tab[9 * n + k] = w;
            } else {
                tab[4 * n + k] = 1.0; tab[5 * n + k] = tab[6 * n + k] = tab[7 * n + k] = tab[8 * n + k] = tab[9 * n + k] = 0.0;
            }
        }
        mhs_status st = upload(ctx, &lv.tab, tab);
        if (st) return st;
        if (dim == 3 && ctx->opt.smoother == MHS_SMOOTH_ZLINE && nz >= 3) {
            // Thomas factors of the z-line matrix T = tridiag(a, D_k, a), a = 1/hz^2 (the same for every line; C25):
            // den_k = D_k - a cp_{k-1}, cp_k = a / den_k;  the kernel multiplies by 1/den_k.
            std::vector<double> zl(2 * (size_t)nz, 0.0);
            const double a = 1.0 / (hz * hz);
            double cprev = 0.0;
            for (int k = 1; k <= nz - 2; ++k) {
                const double den = tab[2 * (size_t)nz + k] - a * cprev;
                if (!(den < 0.0)) return fail(ctx, MHS_ERR_INDEFINITE, "z-line matrix is not negative definite (alpha^2 too large)");
                cprev = a / den;
                zl[k] = cprev;
                zl[(size_t)nz + k] = 1.0 / den;
            }
            if ((st = upload(ctx, &lv.zl, zl))) return st;
        }
        if ((st = alloc_field(ctx, lv, 0, &lv.u))) return st;
        if (!(dim == 3 && l == 0) || ctx->wall_ctx)   // (eq 8 is homogeneous: no right-hand side on the finest 3D level -- unless wall data is lifted into one)
            if ((st = alloc_field(ctx, lv, 2, &lv.rhs))) return st;
        if (!lv.coarsest) {
            if ((st = alloc_field(ctx, lv, 1, &lv.tmp))) return st;
            if ((st = alloc_field(ctx, lv, 3, &lv.r))) return st;
        } else {
            // exact solve on the coarsest level (C9): assemble L on the interior unknowns, invert.
            const int mx = nx - 2, my = ny - 2, mz = dim == 3 ? nz - 2 : 1;
            const long long n = (long long)mx * my * mz;
            if (n > 1024) return fail(ctx, MHS_ERR_GRID, "coarsest level has more than 1024 unknowns; extents must be 2^m*q+1 with small q");
            lv.ncoarse = (int)n;
            std::vector<double> A((size_t)n * n, 0.0);
            for (int k = 0; k < mz; ++k)
                for (int j = 0; j < my; ++j)
                    for (int i = 0; i < mx; ++i) {
                        const int row = i + mx * (j + my * k);
                        const int kk = dim == 3 ? k + 1 : 0;
                        const double cx = c[kk] / (hx * hx), cy = c[kk] / (hy * hy), cz = dim == 3 ? 1.0 / (hz * hz) : 0.0;
                        A[(size_t)row * n + row] = -2.0 * cx - 2.0 * cy - 2.0 * cz + a2;
                        if (i > 0) A[(size_t)row * n + row - 1] = cx;
                        if (i < mx - 1) A[(size_t)row * n + row + 1] = cx;
                        if (j > 0) A[(size_t)row * n + row - mx] = cy;
                        if (j < my - 1) A[(size_t)row * n + row + mx] = cy;
                        if (k > 0) A[(size_t)row * n + row - mx * my] = cz;
                        if (k < mz - 1) A[(size_t)row * n + row + mx * my] = cz;
                    }
            if (!invert_dense((int)n, A)) return fail(ctx, MHS_ERR_INDEFINITE, "coarsest-level operator is singular");
            if ((st = upload(ctx, &lv.ainv, A))) return st;
        }
        Ls.push_back(lv);
        if (lv.coarsest) break;
        // next level: rediscretise with 2h, inject the coefficient (C7)
        std::vector<double> cc((nz - 1) / 2 + 1);
        if (dim == 3) {
            for (size_t K = 0; K < cc.size(); ++K) cc[K] = c[2 * K];
            c = cc;
            nz = (nz - 1) / 2 + 1;
            hz *= 2.0;
        }
        nx = (nx - 1) / 2 + 1; ny = (ny - 1) / 2 + 1;
        hx *= 2.0; hy *= 2.0;
    }
    return MHS_OK;
}

void* field_base(const mhs_ctx* ctx, const Level& lv, void* p) { return (char*)p - (size_t)lv.pad * ctx->es; }

// ---------------------------------------------------------------------------------------------
// V-cycle, reference composition (SURVEY 8(c) "V(u,rhs,l)"): one kernel per component.
// ---------------------------------------------------------------------------------------------
int kc_for(const Level& lv, int l, int what /*0 smooth 1 restrict 2 prolong 3 norm*/)
{
    if (lv.dim == 2) return MHS_KC_BOUNDARY_2D;
    if (l > 0) return MHS_KC_COARSE_3D;
    return what;
}

// z-line Jacobi smoothing (mhs_options.smoother) applies to the 3D hierarchy
bool use_zline(const mhs_ctx* ctx, const Level& lv) { return ctx->opt.smoother == MHS_SMOOTH_ZLINE && lv.dim == 3 && zline_ok(ctx, lv); }

bool use_fast(const mhs_ctx* ctx, const Level& lv)
{
    return !(ctx->opt.flags & MHS_FLAG_REFERENCE_KERNELS) && fast_ok(ctx, lv) && &lv != ctx->ref_level;
}

bool use_zsweep(const mhs_ctx* ctx, const Level& lv)
{
    return !(ctx->opt.flags & (MHS_FLAG_REFERENCE_KERNELS | MHS_FLAG_UNFUSED_KERNELS)) && !mid_level(ctx, lv) && zsweep_ok(ctx, lv) &&
           !(ctx->opt.smoother == MHS_SMOOTH_ZLINE && lv.dim == 3);
}

// A stop rule that vcycle() left to the finest-level restriction and that kernel cannot take: as a launch of its own.
void flush_pending_norm(mhs_ctx* ctx, const Level& lv)
{
    if (ctx->pending_norm <= 0) return;
    const int prev = ctx->cur_kc;
    ctx->cur_kc = lv.dim == 3 ? MHS_KC_NORM_L0 : prev;
    launch_norm_final(ctx, ctx->pending_norm, 1);
    ctx->cur_kc = prev;
    ctx->pending_norm = 0;
}

// residual + full weighting into co.rhs: separable form on big levels, register z-streaming on the others
void restrict_fast(mhs_ctx* ctx, const Level& lv, const void* u, const void* rhs, const Level& co, int reverse, const int* done)
{
    if (!mid_level(ctx, lv) && !(ctx->opt.flags & MHS_FLAG_UNFUSED_KERNELS) && lv.nz >= 5) {
        // no right-hand side (the finest level): the bulk-copy fed kernel (walking down in z, to meet the planes the smoothing
        // pass wrote last while they are still in the L2, measured no different from walking up: 31.7 against 31.0 us at 257^3)
        if (!rhs && !(ctx->opt.flags & MHS_FLAG_LOADED_RESTRICT)) {
            const long long np = ctx->pending_norm;
            if (launch_resid_restrict_ring(ctx, lv, u, co, co.rhs, 0, done, np)) { ctx->pending_norm = 0; return; }
            if (np > 0) {    // could not be folded in after all: the stop rule as a launch of its own, then the restriction
                flush_pending_norm(ctx, lv);
                if (launch_resid_restrict_ring(ctx, lv, u, co, co.rhs, 0, done)) return;
            }
        }
        flush_pending_norm(ctx, lv);
        launch_resid_restrict_sep(ctx, lv, u, rhs, co, co.rhs, reverse, done);
    } else {
        flush_pending_norm(ctx, lv);
        if (rhs && !(ctx->opt.flags & MHS_FLAG_UNFUSED_KERNELS) && resid_restrict_box_ok(ctx, lv)) launch_resid_restrict_box(ctx, lv, u, rhs, co, co.rhs, done);
        else launch_resid_restrict_z(ctx, lv, u, rhs, co, co.rhs, reverse, done);
    }
}

int clus_of(const mhs_ctx* ctx, const std::vector<Level>& Ls) { return Ls[0].dim == 3 ? ctx->clus3 : ctx->clus2; }

// `sweeps` Jacobi sweeps on level l, ping-ponging lv.u <-> lv.tmp.  want_norm: the first sweep also leaves
// the partial sums of ||rhs - L u||^2 of ITS INPUT in ctx->partial (returned count; 0 = not computed).
long long smooth(mhs_ctx* ctx, std::vector<Level>& Ls, int l, int sweeps, const int* done, bool want_norm = false)
{
    Level& lv = Ls[l];
    const void* rhs = lv.rhs /* (finest 3D level: NULL unless wall data is lifted into it) */;
    const bool fast = use_fast(ctx, lv);
    long long npart = 0;
    if (use_zline(ctx, lv)) {    // z-line Jacobi: one tridiagonal solve per (i,j) line and sweep (no norm by-product)
        for (int s = 0; s < sweeps; ++s) {
            Scope sc(ctx, kc_for(lv, l, 0));
            launch_zline(ctx, lv, lv.u, rhs, lv.tmp, done);
            std::swap(lv.u, lv.tmp);
            if (lv.dim == 3 && l == 0) ctx->prof.sweeps_l0 += 1;
        }
        return 0;
    }
    if (use_zsweep(ctx, lv)) {   // temporally blocked: two sweeps per pass over the iterate
        for (int s = 0; s < sweeps;) {
            const int S = std::min(2, sweeps - s);
            Scope sc(ctx, kc_for(lv, l, 0));
            const int n = launch_zsweep(ctx, lv, lv.u, rhs, lv.tmp, S, false, want_norm && s == 0, done);
            if (want_norm && s == 0) npart = n;
            std::swap(lv.u, lv.tmp);
            if (lv.dim == 3 && l == 0) ctx->prof.sweeps_l0 += S;
            s += S;
        }
        return npart;
    }
    for (int s = 0; s < sweeps; ++s) {
        Scope sc(ctx, kc_for(lv, l, 0));
        if (fast && l > 0 && rhs && sweeps - s >= 2 && !(want_norm && s == 0) && smooth2_node_ok(ctx, lv) &&
            !(ctx->opt.flags & MHS_FLAG_UNFUSED_KERNELS)) {
            launch_smooth2_node(ctx, lv, lv.u, rhs, lv.tmp, done);      // two sweeps, one launch (small levels)
            std::swap(lv.u, lv.tmp);
            ++s;
            continue;
        }
        if (fast) {
            const long long n = launch_smooth_z(ctx, lv, lv.u, rhs, lv.tmp, (want_norm && s == 0) ? 1 : 0, ctx->dir, done);
            if (want_norm && s == 0) npart = n;
            ctx->dir ^= 1;
        } else {
            launch_smooth_ref(ctx, lv, lv.u, rhs, lv.tmp, done);
        }
        std::swap(lv.u, lv.tmp);
        if (lv.dim == 3 && l == 0) ctx->prof.sweeps_l0 += 1;
    }
    return npart;
}

// Partial sums of ||rhs - L u||^2 on level l -> ctx->partial; returns their count.
long long resnorm_partials(mhs_ctx* ctx, std::vector<Level>& Ls, int l, const int* done)
{
    Level& lv = Ls[l];
    const void* rhs = lv.rhs /* (finest 3D level: NULL unless wall data is lifted into it) */;
    Scope sc(ctx, kc_for(lv, l, 3));
    if (use_fast(ctx, lv)) return launch_smooth_z(ctx, lv, lv.u, rhs, nullptr, 2, 0, done);
    return launch_resnorm_partial_ref(ctx, lv, lv.u, rhs, done);
}

void norm_final(mhs_ctx* ctx, const Level& lv, int l, long long n, int mode)
{
    Scope sc(ctx, kc_for(lv, l, 3));
    launch_norm_final(ctx, n, mode);
}

// One V-cycle from level l (SURVEY 8(c) "V(u,rhs,l)").  Levels >= 1 start from u = 0.  At l == 0 with
// fuse_norm the norm of the incoming iterate's residual is taken inside the first pre-sweep and the
// stop rule (norm_final mode 1) is evaluated right after it, before the rest of the cycle is allowed to run.
// cont (full-multigrid start, C26): level l >= 1 CONTINUES from the iterate in lv.u, whose bottom plane carries Dirichlet
// data -- general kernels only on this level (no zero-guess shortcuts, not the cluster kernel, whose shared-memory levels
// have zero walls); the levels below it are ordinary coarse-grid corrections.
void vcycle(mhs_ctx* ctx, std::vector<Level>& Ls, int l, const int* done, bool fuse_norm = false, bool cont = false)
{
    Level& lv = Ls[l];
    const void* rhs = lv.rhs /* (finest 3D level: NULL unless wall data is lifted into it) */;
    if (l >= clus_of(ctx, Ls) && !lv.coarsest && !cont) {   // this level and everything below it: one cluster-kernel launch
        Scope sc(ctx, kc_for(lv, l, 0));
        launch_cluster(ctx, Ls, l, l == 0 ? 1 : 0, done);
        return;
    }
    if (lv.coarsest) {
        Scope sc(ctx, kc_for(lv, l, 0));
        launch_coarse_solve(ctx, lv, lv.u, rhs, done);
        return;
    }
    Level& co = Ls[l + 1];
    const bool fast = use_fast(ctx, lv);
    int n_pre = ctx->opt.n_pre;
    const bool zs = use_zsweep(ctx, lv);
    if (l > 0 && !cont) {  // zero initial guess
        Scope sc(ctx, kc_for(lv, l, 0));
        if (use_zline(ctx, lv)) {
            cudaMemsetAsync(field_base(ctx, lv, lv.u), 0, (size_t)lv.alloc * ctx->es, ctx->stream);
        } else if (zs && n_pre >= 1) {
            // the first sweep from zero is u = (omega/D) rhs: folded into the first temporally blocked pass
            const int S = std::min(2, n_pre);
            launch_zsweep(ctx, lv, nullptr, rhs, lv.u, S, true, false, done);
            n_pre -= S;
        } else if (fast && n_pre >= 2) {
            // the first two sweeps from zero in one pass over rhs (sweep 1, u = (omega/D) rhs, is never stored)
            launch_smooth_z(ctx, lv, nullptr, rhs, lv.u, 3, ctx->dir, done);
            ctx->dir ^= 1;
            n_pre -= 2;
        } else if (fast && n_pre >= 1) {
            launch_scale_rhs(ctx, lv, rhs, lv.u, done);  // first sweep from zero: u = (omega/D) rhs
            n_pre -= 1;
        } else {
            cudaMemsetAsync(field_base(ctx, lv, lv.u), 0, (size_t)lv.alloc * ctx->es, ctx->stream);
        }
    }
    if (fuse_norm && l == 0) {
        const int first = zs ? std::min(2, n_pre) : 1;
        // Launched behind `done` like every other kernel of the cycle: in the unit that finds the stop rule met the flag is
        // still down when this pass starts (the flag is raised by the norm_final that follows it), so it runs and leaves the
        // norm; in the speculative units issued after that one it is skipped.  (Launched unconditionally it would, in those
        // later units and for an odd number of ping-pong passes per cycle, write into the buffer that holds the final iterate.)
        const long long np = smooth(ctx, Ls, l, first, done, true);
        // The stop rule: a one-block kernel of its own -- or, when the restriction follows at once (no pre-smoothing pass
        // left, which would overwrite the iterate) and is the bulk-copy fed kernel, folded into that kernel's CTA 0
        // (restrict_fast): one dependent launch less per cycle, ~4 us at 257^3.
        if (n_pre - first == 0 && fast && !rhs && ctx->opt.profile < 2 && !(ctx->opt.flags & MHS_FLAG_NO_FOLDED_NORM)) ctx->pending_norm = np;
        else norm_final(ctx, lv, l, np, 1);
        smooth(ctx, Ls, l, n_pre - first, done);
    } else {
        smooth(ctx, Ls, l, n_pre, done);
    }
    {
        Scope sc(ctx, kc_for(lv, l, 1));
        if (fast) {
            restrict_fast(ctx, lv, lv.u, rhs, co, ctx->dir, done);
            ctx->dir ^= 1;
        } else {
            launch_residual_ref(ctx, lv, lv.u, rhs, lv.r, done);
            launch_restrict_ref(ctx, lv, lv.r, co, co.rhs, done);
        }
    }
    vcycle(ctx, Ls, l + 1, done);
    int n_post = ctx->opt.n_post;
    bool fused_prolong = false;
    if (zs && n_post >= 1 && !(ctx->opt.flags & MHS_FLAG_SEPARATE_PROLONG)) {
        // prolongation + correction folded into the first post-smoothing pass (no pass of its own over u)
        Scope sc(ctx, kc_for(lv, l, 2));
        const int S = std::min(2, n_post);
        fused_prolong = launch_zsweep_prolong(ctx, lv, lv.u, rhs, lv.tmp, S, co, co.u, done);
        if (fused_prolong) {
            std::swap(lv.u, lv.tmp);
            if (lv.dim == 3 && l == 0) { ctx->prof.sweeps_l0 += S; ctx->prof.fused_prolong_l0 += 1; }
            n_post -= S;
        }
    }
    if (!fused_prolong) {
        Scope sc(ctx, kc_for(lv, l, 2));
        if (fast) {
            launch_prolong_v(ctx, lv, lv.u, co, co.u, ctx->dir, done);
            ctx->dir ^= 1;
        } else {
            launch_prolong_ref(ctx, lv, lv.u, co, co.u, done);
        }
    }
    smooth(ctx, Ls, l, n_post, done);
}

// Report a finished solve loop from the control block read back into ctx->ctl_host.
mhs_status finish_cycles(mhs_ctx* ctx, double tol, mhs_solve_info* info)
{
    const Ctl* h = ctx->ctl_host;
    if (info) {
        info->cycles = h->cycles;
        info->r0 = h->r0;
        info->r_final = h->cycles > 0 ? h->r_last : h->r0;
        info->stagnated = h->stagnated;
        memset(info->history, 0, sizeof info->history);
        memcpy(info->history, h->hist, sizeof(double) * std::min(h->cycles, MHS_HISTORY_LEN));
    }
    if (h->nan_seen) return fail(ctx, MHS_ERR_INDEFINITE, "residual norm is not finite (divergence: alpha^2 too large for the coarse grids?)");
    if (!(h->r_last <= tol * h->r0) && !h->stagnated) return fail(ctx, MHS_ERR_NOT_CONVERGED, "max_cycles reached before the tolerance");
    return MHS_OK;
}

// Solve loop shared by the 2D and 3D drivers.  Unit q = [norm of iterate q-1 -> stop rule] + [V-cycle q];
// units run speculatively in chunks behind the device-side stop flag and the host reads the control block
// once per chunk.  The stop rule (C10) is exact: once the flag is up every later kernel returns at once, and
// the only kernel that has already run in the stopping unit -- the first pre-sweep, which carries the norm --
// writes the ping-pong buffer, never the iterate.  iter_buf[q] remembers which buffer holds iterate q.
mhs_status run_cycles(mhs_ctx* ctx, std::vector<Level>& Ls, double tol, int max_cycles, double r0_known,
                      mhs_solve_info* info)
{
    if (max_cycles < 1) return fail(ctx, MHS_ERR_INVALID_ARG, "max_cycles must be >= 1");
    Ctl* h = ctx->ctl_host;
    memset(h, 0, sizeof(Ctl));
    h->max_cycles = max_cycles;
    h->tol = tol;
    h->r0 = r0_known;
    h->stag_on = ctx->es == 4;
    CK(cudaMemcpyAsync(ctx->ctl, h, sizeof(Ctl), cudaMemcpyHostToDevice, ctx->stream));
    Level& l0 = Ls[0];
    const int* done = &ctx->ctl->done;
    const bool sync_each = (ctx->opt.flags & MHS_FLAG_SYNC_EACH_CYCLE) != 0;
    if (clus_of(ctx, Ls) == 0 && !l0.coarsest && !sync_each) {
        // The finest level is itself a cluster level: the whole solve loop runs in ONE kernel launch.
        {
            Scope sc(ctx, kc_for(l0, 0, 0));
            launch_cluster(ctx, Ls, 0, 2, nullptr);
        }
        { mhs_status rs = read_ctl(ctx); if (rs) return rs; }
        drain_events(ctx);
        CK(cudaGetLastError());
        if ((h->cycles * (ctx->opt.n_pre + ctx->opt.n_post)) & 1) std::swap(l0.u, l0.tmp);
        return finish_cycles(ctx, tol, info);
    }
    const bool fuse = use_fast(ctx, l0) && ctx->opt.n_pre >= 1 && !l0.coarsest && clus_of(ctx, Ls) > 0 && !use_zline(ctx, l0);
    std::vector<void*> iter_buf(1, l0.u);
    int issued = 0;
    bool trailing = false;
    while (true) {
        // How many units to issue before the next read-back: 4 to start with, then the number the observed
        // convergence factor predicts are still needed (+1: a cycle's norm is taken by the unit after it),
        // so that hardly any speculative unit is wasted.  Purely a scheduling choice: results do not depend on it.
        int want = 4;
        if (h->cycles >= 2 && h->cycles <= MHS_HISTORY_LEN) {
            const double rl = h->hist[h->cycles - 1], rp = h->hist[h->cycles - 2];
            const double target = tol * h->r0;
            if (rl > 0.0 && rp > rl && target > 0.0 && rl > target) {
                const double need = std::ceil(std::log(target / rl) / std::log(rl / rp));
                want = (int)std::min(16.0, std::max(1.0, h->cycles + need + 1 - issued));
            }
        }
        const int n = std::min(sync_each ? 1 : want, max_cycles - issued);
        for (int q = 0; q < n; ++q) {
            if (fuse) {
                vcycle(ctx, Ls, 0, done, true);
            } else {
                const long long np = resnorm_partials(ctx, Ls, 0, done);
                norm_final(ctx, l0, 0, np, 1);
                vcycle(ctx, Ls, 0, done);
            }
            iter_buf.push_back(l0.u);
        }
        issued += n;
        if (issued >= max_cycles) {  // norm of the last iterate
            const long long np = resnorm_partials(ctx, Ls, 0, done);
            norm_final(ctx, l0, 0, np, 1);
            trailing = true;
        }
        { mhs_status rs = read_ctl(ctx); if (rs) return rs; }
        if (h->done || trailing) break;
    }
    drain_events(ctx);
    CK(cudaGetLastError());
    // put the final iterate back under the name `u`
    if (l0.tmp && h->cycles >= 0 && h->cycles < (int)iter_buf.size()) {
        void* fin = iter_buf[h->cycles];
        if (fin != l0.u) std::swap(l0.u, l0.tmp);
    }
    return finish_cycles(ctx, tol, info);
}

// pending host copies (mhs_fields_host_async) read the staging buffer: later work on the main stream that overwrites it waits
mhs_status stage_fence(mhs_ctx* ctx)
{
    if (ctx->copy_pending) CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_copied, 0));
    return MHS_OK;
}

mhs_status ensure_stage(mhs_ctx* ctx, size_t bytes)
{
    if (ctx->stage_bytes >= bytes) return MHS_OK;
    if (ctx->copy_pending) { CK(cudaEventSynchronize(ctx->ev_copied)); ctx->copy_pending = false; }
    if (ctx->stage) cudaFree(ctx->stage);
    ctx->stage = nullptr; ctx->stage_bytes = 0;
    CK(cudaMalloc(&ctx->stage, bytes));
    ctx->stage_bytes = bytes;
    return MHS_OK;
}

std::vector<Level>* hierarchy(mhs_ctx* ctx, int dim) { return dim == 3 ? &ctx->L3 : dim == 2 ? &ctx->L2 : nullptr; }

mhs_status check_level(mhs_ctx* ctx, int dim, int level, std::vector<Level>** Ls)
{
    *Ls = hierarchy(ctx, dim);
    if (!*Ls) return fail(ctx, MHS_ERR_INVALID_ARG, "dim must be 2 or 3");
    if (level < 0 || level >= (int)(*Ls)->size()) return fail(ctx, MHS_ERR_INVALID_ARG, "no such level");
    return MHS_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

void mhs_default_options(mhs_options* o)
{
    if (!o) return;
    memset(o, 0, sizeof *o);
    o->dtype = MHS_F64;
    o->omega = 2.0 / 3.0;
    o->n_pre = 2; o->n_post = 2;
    o->max_levels = 0;
    o->boundary_tol = 1e-10;
    o->boundary_max_cycles = 100;
    o->mu0 = 0.5; o->g = 1.0;
}

const char* mhs_status_string(mhs_status s)
{
    switch (s) {
        case MHS_OK: return "MHS_OK";
        case MHS_ERR_INVALID_ARG: return "MHS_ERR_INVALID_ARG";
        case MHS_ERR_GRID: return "MHS_ERR_GRID";
        case MHS_ERR_NOT_ELLIPTIC: return "MHS_ERR_NOT_ELLIPTIC";
        case MHS_ERR_INDEFINITE: return "MHS_ERR_INDEFINITE";
        case MHS_ERR_STATE: return "MHS_ERR_STATE";
        case MHS_ERR_NOT_CONVERGED: return "MHS_ERR_NOT_CONVERGED";
        case MHS_ERR_CUDA: return "MHS_ERR_CUDA";
        case MHS_ERR_OOM: return "MHS_ERR_OOM";
    }
    return "MHS_ERR_?";
}

const char* mhs_kernel_class_name(int kc)
{
    static const char* n[MHS_KC_COUNT] = {"smooth_l0", "restrict_l0", "prolong_l0", "norm_l0",
                                          "coarse_3d", "boundary_2d", "fields", "pack"};
    return (kc >= 0 && kc < MHS_KC_COUNT) ? n[kc] : "?";
}

const char* mhs_last_error(const mhs_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

mhs_status mhs_create(const mhs_grid* grid, double alpha, const double* f_profile, const mhs_bc* bc,
                      const mhs_options* opts, mhs_ctx** out)
{
    if (!grid || !out) return MHS_ERR_INVALID_ARG;
    *out = nullptr;
    mhs_ctx* ctx = new (std::nothrow) mhs_ctx();
    if (!ctx) return MHS_ERR_OOM;
    // from here on errors are reported through a context the caller can query and must destroy
    *out = ctx;
    ctx->grid = *grid;
    if (opts) ctx->opt = *opts; else mhs_default_options(&ctx->opt);
    ctx->alpha = alpha;
    const mhs_options& o = ctx->opt;
    if (o.dtype != MHS_F32 && o.dtype != MHS_F64) return fail(ctx, MHS_ERR_INVALID_ARG, "dtype must be MHS_F32 or MHS_F64");
    ctx->es = o.dtype == MHS_F64 ? 8 : 4;
    ctx->stream = (cudaStream_t)o.stream;
    if (bc) {
        for (int v : {bc->sides, bc->top})
            if (v != MHS_BC_DIRICHLET_ZERO && v != MHS_BC_DIRICHLET_DATA)
                return fail(ctx, MHS_ERR_INVALID_ARG, "mhs_bc: MHS_BC_DIRICHLET_ZERO (P = 0, PAPER.md:96) or MHS_BC_DIRICHLET_DATA (P given, mhs_set_wall_data)");
        ctx->bc_sides = bc->sides; ctx->bc_top = bc->top;
        ctx->wall_ctx = grid->nz > 1 && (bc->sides == MHS_BC_DIRICHLET_DATA || bc->top == MHS_BC_DIRICHLET_DATA);
        if (ctx->wall_ctx && (ctx->opt.smoother != MHS_SMOOTH_JACOBI || ctx->opt.fmg_cycles != 0))
            return fail(ctx, MHS_ERR_INVALID_ARG, "MHS_BC_DIRICHLET_DATA needs the point-Jacobi smoother and fmg_cycles = 0");
    }
    if (!(o.omega > 0.0 && o.omega <= 1.0) || o.n_pre < 0 || o.n_post < 0 || o.n_pre + o.n_post < 1 || o.max_levels < 0 ||
        !(o.mu0 > 0.0) || o.g == 0.0 || o.boundary_max_cycles < 1 || !(grid->Lx > 0 && grid->Ly > 0 && grid->Lz > 0) ||
        (o.smoother != MHS_SMOOTH_JACOBI && o.smoother != MHS_SMOOTH_ZLINE) || o.fmg_cycles < 0)
        return fail(ctx, MHS_ERR_INVALID_ARG, "invalid option value");
    const int ext[3] = {grid->nx, grid->ny, grid->nz};
    const bool only2d = grid->nz == 1;   // boundary-only context: eq (11) on the plane, no interior (mhs.h, mhs_create)
    for (int a = 0; a < (only2d ? 2 : 3); ++a)
        if (ext[a] < 3 || ((ext[a] - 1) & 1))
            return fail(ctx, MHS_ERR_GRID, "every extent must be 2^m*q+1 with m >= 1 (an even number >= 2 of intervals); nz = 1 = 2D only");
    const int nz = grid->nz;
    ctx->f.assign(nz, 0.0);
    if (f_profile) ctx->f.assign(f_profile, f_profile + nz);
    for (int k = 0; k < nz; ++k)
        if (!(1.0 + ctx->f[k] > 0.0)) return fail(ctx, MHS_ERR_NOT_ELLIPTIC, "1 + f(z_k) <= 0: eq (8) is not elliptic (PAPER.md:70)");
    ctx->p_b.assign(nz, 0.0); ctx->rho_b.assign(nz, 0.0); ctx->dfdz.assign(nz, 0.0);
    if (o.p_b) ctx->p_b.assign(o.p_b, o.p_b + nz);
    if (o.rho_b) ctx->rho_b.assign(o.rho_b, o.rho_b + nz);
    const double hz = grid->Lz / (nz - 1);
    if (o.dfdz) ctx->dfdz.assign(o.dfdz, o.dfdz + nz);
    else if (!only2d) {  // C14: central differences of the samples, one-sided second order at both ends
        const std::vector<double>& f = ctx->f;
        for (int k = 1; k < nz - 1; ++k) ctx->dfdz[k] = (f[k + 1] - f[k - 1]) / (2.0 * hz);
        ctx->dfdz[0] = (-3.0 * f[0] + 4.0 * f[1] - f[2]) / (2.0 * hz);
        ctx->dfdz[nz - 1] = (3.0 * f[nz - 1] - 4.0 * f[nz - 2] + f[nz - 3]) / (2.0 * hz);
    }
    ctx->opt.p_b = ctx->opt.rho_b = ctx->opt.dfdz = nullptr;  // the caller's arrays are not kept

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(ctx, MHS_ERR_CUDA, "no CUDA device: libmhs_b200 has no CPU fallback");
    }
    mhs_status st;
    if (!only2d && (st = build_hierarchy(ctx, 3, ctx->L3))) return st;
    if ((st = build_hierarchy(ctx, 2, ctx->L2))) return st;
    if (!only2d && ctx->L3.size() < 2) return fail(ctx, MHS_ERR_GRID, "the 3D hierarchy needs at least two levels (>= 4 intervals per axis, max_levels != 1)");

    std::vector<double> ft(4 * (size_t)nz);
    for (int k = 0; k < nz; ++k) {
        ft[k] = -ctx->f[k];            // xi = -f   (C1)
        ft[nz + k] = -ctx->dfdz[k];    // xi'
        ft[2 * nz + k] = ctx->p_b[k];
        ft[3 * nz + k] = ctx->rho_b[k];
    }
    if ((st = upload(ctx, &ctx->prof_tab, ft))) return st;
    {
        int dev = 0;
        cudaDeviceProp pr;
        CK(cudaGetDevice(&dev));
        CK(cudaGetDeviceProperties(&pr, dev));
        ctx->num_sms = pr.multiProcessorCount;
        ctx->device = dev;
        ctx->debug = getenv("MHS_DEBUG") != nullptr;
        ctx->no_align = getenv("MHS_NO_ALIGN") != nullptr;
        if (const char* e = getenv("MHS_MID_PTS")) ctx->mid_pts = atoll(e);
        if (const char* e = getenv("MHS_S2_PTS")) ctx->s2_pts = atoll(e);
        if (const char* e = getenv("MHS_RB_PTS")) ctx->rb_pts = atoll(e);
        if (const char* e = getenv("MHS_CL3_PTS")) ctx->cl3_pts = atoll(e);
    }
    const bool ref = (ctx->opt.flags & MHS_FLAG_REFERENCE_KERNELS) != 0;
    const bool ref3 = ref || ctx->opt.smoother == MHS_SMOOTH_ZLINE;   // (the cluster kernel smooths with point Jacobi)
    ctx->tail3 = (ref3 || only2d) ? (int)ctx->L3.size() : tail_start(ctx, ctx->L3, 216 * 1024);
    ctx->tail2 = ref ? (int)ctx->L2.size() : tail_start(ctx, ctx->L2, 216 * 1024);
    ctx->clus3 = (ref3 || only2d) ? (int)ctx->L3.size() : cluster_start(ctx, ctx->L3, ctx->tail3);
    ctx->clus2 = ref ? (int)ctx->L2.size() : cluster_start(ctx, ctx->L2, ctx->tail2);
    if (!ref) ctx->cluster_max = cluster_max_size(ctx);
    ctx->npartial = std::max<long long>(64, resnorm_partial_capacity(ctx->L2[0]));
    if (!only2d) ctx->npartial = std::max(ctx->npartial, resnorm_partial_capacity(ctx->L3[0]));
    for (const Level& lv : ctx->L3) ctx->npartial = std::max(ctx->npartial, smooth_z_partial_capacity(ctx, lv));
    ctx->npartial = std::max<long long>(ctx->npartial, 4 * ctx->num_sms);
    if (ctx->wall_ctx) {   // wall data W and a dense scratch copy of P for mhs_fields, both N elements, W = 0 until mhs_set_wall_data
        const size_t nb = (size_t)ctx->L3[0].npts() * ctx->es;
        CK(cudaMalloc(&ctx->wall, nb));
        CK(cudaMemset(ctx->wall, 0, nb));
        CK(cudaMalloc(&ctx->dense_P, nb));
    }
    CK(cudaMalloc((void**)&ctx->partial, sizeof(double) * (size_t)ctx->npartial));
    CK(cudaMalloc((void**)&ctx->ctl, sizeof(Ctl)));
    CK(cudaMemset(ctx->ctl, 0, sizeof(Ctl)));
    CK(cudaHostAlloc((void**)&ctx->ctl_host, sizeof(Ctl), cudaHostAllocMapped));   // (unified addressing: usable on the device as is)
    CK(cudaMalloc(&ctx->bz_stage, (size_t)grid->nx * grid->ny * ctx->es));
    CK(cudaDeviceSynchronize());
    return MHS_OK;
}

void mhs_destroy(mhs_ctx* ctx)
{
    if (!ctx) return;
    if (ctx->stream || !ctx->L3.empty()) cudaStreamSynchronize(ctx->stream);
    for (std::vector<Level>* Ls : {&ctx->L3, &ctx->L2})
        for (Level& lv : *Ls) {
            for (void* p : lv.raw) if (p) cudaFree(p);
            if (lv.tab) cudaFree(lv.tab);
            if (lv.ainv) cudaFree(lv.ainv);
            if (lv.zl) cudaFree(lv.zl);
        }
    if (ctx->prof_tab) cudaFree(ctx->prof_tab);
    if (ctx->partial) cudaFree(ctx->partial);
    if (ctx->ctl) cudaFree(ctx->ctl);
    if (ctx->ctl_host) cudaFreeHost(ctx->ctl_host);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    if (ctx->ev_fields) cudaEventDestroy(ctx->ev_fields);
    if (ctx->ev_copied) cudaEventDestroy(ctx->ev_copied);
    if (ctx->stage) cudaFree(ctx->stage);
    if (ctx->bz_stage) cudaFree(ctx->bz_stage);
    if (ctx->wall) cudaFree(ctx->wall);
    if (ctx->dense_P) cudaFree(ctx->dense_P);
    for (const Ev& e : ctx->ev_pending) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    delete ctx;
}

mhs_status mhs_solve_boundary(mhs_ctx* ctx, const void* Bz0, mhs_solve_info* info)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (!Bz0) return fail(ctx, MHS_ERR_INVALID_ARG, "Bz0 is NULL");
    if (ctx->L2.empty()) return fail(ctx, MHS_ERR_STATE, "context was not created successfully");
    const bool have3 = !ctx->L3.empty();
    Level& l3 = have3 ? ctx->L3[0] : ctx->L2[0];   // (a 2D-only context has no interior to fill)
    Level& l2 = ctx->L2[0];
    {
        Scope sc(ctx, MHS_KC_PACK);
        // step 1: P = 0 everywhere
        if (have3) {
            CK(cudaMemsetAsync(field_base(ctx, l3, l3.u), 0, (size_t)l3.alloc * ctx->es, ctx->stream));
            CK(cudaMemsetAsync(field_base(ctx, l3, l3.tmp), 0, (size_t)l3.alloc * ctx->es, ctx->stream));
        }
        CK(cudaMemsetAsync(field_base(ctx, l2, l2.u), 0, (size_t)l2.alloc * ctx->es, ctx->stream));
        if (l2.tmp) CK(cudaMemsetAsync(field_base(ctx, l2, l2.tmp), 0, (size_t)l2.alloc * ctx->es, ctx->stream));
        launch_pack(ctx, l2, Bz0, l2.rhs, true, true);  // rhs2 = -Bz0 at interior nodes (eq 11)
    }
    ctx->have_boundary = false;
    ctx->have_r0 = false;
    // step 2
    mhs_status st = run_cycles(ctx, ctx->L2, ctx->opt.boundary_tol, ctx->opt.boundary_max_cycles, 0.0, info);
    if (st != MHS_OK && st != MHS_ERR_NOT_CONVERGED) return st;
    if (have3) {
        Scope sc(ctx, MHS_KC_PACK);
        // P(:,:,0) = P0, in both ping-pong buffers of the finest 3D level (same in-plane layout)
        CK(cudaMemcpyAsync(l3.u, ctx->L2[0].u, (size_t)l2.sp * ctx->es, cudaMemcpyDeviceToDevice, ctx->stream));
        CK(cudaMemcpyAsync(l3.tmp, ctx->L2[0].u, (size_t)l2.sp * ctx->es, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    ctx->have_boundary = have3;
    ctx->fmg_pending = have3;
    return st;
}

mhs_status mhs_solve_boundary_host(mhs_ctx* ctx, const void* Bz0_host, mhs_solve_info* info)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (!Bz0_host) return fail(ctx, MHS_ERR_INVALID_ARG, "Bz0 is NULL");
    // (a buffer of its own: the big staging buffer may still be feeding the host copies of the previous step's fields)
    const size_t bytes = (size_t)ctx->grid.nx * ctx->grid.ny * ctx->es;
    CK(cudaMemcpyAsync(ctx->bz_stage, Bz0_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    return mhs_solve_boundary(ctx, ctx->bz_stage, info);
}

// Residual norm of the current level-0 iterate of a hierarchy, read back (one stream synchronisation).
static mhs_status resnorm_now(mhs_ctx* ctx, std::vector<Level>& Ls, double* out)
{
    const long long np = resnorm_partials(ctx, Ls, 0, nullptr);
    norm_final(ctx, Ls[0], 0, np, 2);
    mhs_status rs = read_ctl(ctx);
    if (rs) return rs;
    drain_events(ctx);
    *out = ctx->ctl_host->r_last;
    return MHS_OK;
}

// Full-multigrid start (mhs_options.fmg_cycles; reading C26): replaces the interior of L3[0].u by the FMG iterate.
// Level l carries the bottom data by injection; coarsest level: exact solve; level l < coarsest: trilinear interpolation
// of the level below (whose bottom plane is then cleared again: below this point it only ever holds coarse-grid
// corrections) + fmg_cycles V-cycles that continue from it.
static mhs_status fmg_start(mhs_ctx* ctx)
{
    std::vector<Level>& Ls = ctx->L3;
    const int n = (int)Ls.size();
    Scope sc(ctx, MHS_KC_COARSE_3D);
    for (int l = 1; l < n; ++l) {
        Level& lv = Ls[l];
        CK(cudaMemsetAsync(field_base(ctx, lv, lv.u), 0, (size_t)lv.alloc * ctx->es, ctx->stream));
        if (lv.tmp) CK(cudaMemsetAsync(field_base(ctx, lv, lv.tmp), 0, (size_t)lv.alloc * ctx->es, ctx->stream));
        CK(cudaMemsetAsync(field_base(ctx, lv, lv.rhs), 0, (size_t)lv.alloc * ctx->es, ctx->stream));
        launch_inject_bottom(ctx, Ls[0], Ls[0].u, lv, 1 << l, lv.u, lv.tmp);
    }
    {
        Level& lc = Ls[n - 1];
        launch_bottom_rhs(ctx, lc, lc.u, lc.rhs);
        launch_coarse_solve(ctx, lc, lc.u, lc.rhs, nullptr);
        CK(cudaMemsetAsync(field_base(ctx, lc, lc.rhs), 0, (size_t)lc.alloc * ctx->es, ctx->stream));
    }
    for (int l = n - 2; l >= 0; --l) {
        Level& lv = Ls[l];
        Level& co = Ls[l + 1];
        // interior <- 0 (planes 1 .. of both buffers' current iterate), then u += P u_coarse: the interpolation itself
        CK(cudaMemsetAsync((char*)lv.u + (size_t)lv.sp * ctx->es, 0, (size_t)lv.sp * (lv.nz - 1) * ctx->es, ctx->stream));
        if (use_fast(ctx, lv)) launch_prolong_v(ctx, lv, lv.u, co, co.u, 0, nullptr);
        else launch_prolong_ref(ctx, lv, lv.u, co, co.u, nullptr);
        // the level below goes back to zero walls
        CK(cudaMemsetAsync(co.u, 0, (size_t)co.sp * ctx->es, ctx->stream));
        if (co.tmp) CK(cudaMemsetAsync(co.tmp, 0, (size_t)co.sp * ctx->es, ctx->stream));
        // (levels the cluster kernel normally runs are tiny: the one-thread-per-node kernels serve them here)
        if (l > 0 && l >= ctx->clus3) ctx->ref_level = &lv;
        for (int q = 0; q < ctx->opt.fmg_cycles; ++q) vcycle(ctx, Ls, l, nullptr, false, l > 0);
        ctx->ref_level = nullptr;
    }
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_solve_interior(mhs_ctx* ctx, double tol, int max_cycles, mhs_solve_info* info)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "context was not created successfully");
    if (!(tol >= 0.0)) return fail(ctx, MHS_ERR_INVALID_ARG, "tol must be >= 0");
    if (!ctx->have_boundary) return fail(ctx, MHS_ERR_STATE, "mhs_solve_interior before a successful mhs_solve_boundary / mhs_set_potential");
    mhs_solve_info local;
    if (!info) info = &local;
    if (ctx->opt.fmg_cycles > 0 && ctx->fmg_pending) {
        ctx->fmg_pending = false;
        // r0 is the residual norm of the iterate the solve starts from by the paper's procedure (zero interior),
        // taken before the full-multigrid start replaces that interior
        double r0 = 0.0, r1 = 0.0;
        mhs_status fs = resnorm_now(ctx, ctx->L3, &r0);
        if (fs) return fs;
        if ((fs = fmg_start(ctx))) return fs;
        if ((fs = resnorm_now(ctx, ctx->L3, &r1))) return fs;
        ctx->have_r0 = r0 > 0.0;
        ctx->r0_interior = r0;
        if (!(r1 == r1) || std::isinf(r1)) return fail(ctx, MHS_ERR_INDEFINITE, "residual norm is not finite after the full-multigrid start");
        if (r1 <= tol * r0) {   // the FMG iterate already meets the tolerance: no ordinary cycle
            memset(info, 0, sizeof *info);
            info->r0 = r0; info->r_final = r1;
            return MHS_OK;
        }
    }
    mhs_status st = run_cycles(ctx, ctx->L3, tol, max_cycles, ctx->have_r0 ? ctx->r0_interior : 0.0, info);
    ctx->fmg_pending = false;
    if (st == MHS_OK || st == MHS_ERR_NOT_CONVERGED) {
        ctx->have_r0 = info->r0 > 0.0;
        ctx->r0_interior = info->r0;
    }
    return st;
}

mhs_status mhs_solve_batch(mhs_ctx* ctx, int nb, const void* Bz0, double tol, int max_cycles, void* P, void* B, void* p, void* rho,
                           mhs_solve_info* infos)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (nb < 0 || (nb > 0 && !Bz0)) return fail(ctx, MHS_ERR_INVALID_ARG, "nb must be >= 0 and Bz0 non-NULL");
    const size_t es = (size_t)ctx->es, n2 = (size_t)ctx->grid.nx * ctx->grid.ny, N = (size_t)ctx->L3[0].npts();
    bool all_converged = true;
    for (int b = 0; b < nb; ++b) {
        mhs_status st = mhs_solve_boundary(ctx, (const char*)Bz0 + (size_t)b * n2 * es, nullptr);
        if (st != MHS_OK && st != MHS_ERR_NOT_CONVERGED) return st;
        st = mhs_solve_interior(ctx, tol, max_cycles, infos ? infos + b : nullptr);
        if (st == MHS_ERR_NOT_CONVERGED) all_converged = false;
        else if (st != MHS_OK) return st;
        if (P && (st = mhs_get_potential(ctx, (char*)P + (size_t)b * N * es))) return st;
        if (B || p || rho)
            if ((st = mhs_fields(ctx, B ? (char*)B + (size_t)b * 3 * N * es : nullptr, p ? (char*)p + (size_t)b * N * es : nullptr,
                                 rho ? (char*)rho + (size_t)b * N * es : nullptr)))
                return st;
    }
    if (!all_converged) return fail(ctx, MHS_ERR_NOT_CONVERGED, "max_cycles reached before the tolerance for at least one member of the batch");
    return MHS_OK;
}

mhs_status mhs_get_potential(mhs_ctx* ctx, void* P)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!P) return fail(ctx, MHS_ERR_INVALID_ARG, "P is NULL");
    Scope sc(ctx, MHS_KC_PACK);
    launch_unpack(ctx, ctx->L3[0], ctx->L3[0].u, P);
    if (ctx->wall_ctx) launch_wall_add(ctx, ctx->L3[0], ctx->wall, P);   // P = P_h + W
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_set_wall_data(mhs_ctx* ctx, const void* G)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (!ctx->wall_ctx) return fail(ctx, MHS_ERR_STATE, "mhs_set_wall_data on a context created without MHS_BC_DIRICHLET_DATA");
    if (!G) return fail(ctx, MHS_ERR_INVALID_ARG, "G is NULL");
    Scope sc(ctx, MHS_KC_PACK);
    Level& l0 = ctx->L3[0];
    launch_wall_take(ctx, l0, ctx->bc_sides == MHS_BC_DIRICHLET_DATA, ctx->bc_top == MHS_BC_DIRICHLET_DATA, G, ctx->wall);
    launch_wall_rhs(ctx, l0, ctx->wall, l0.rhs);   // (only interior nodes are written; the rest of rhs0 stays zero)
    ctx->have_r0 = false;                          // r0 belongs to the problem: the next solve takes it afresh
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_get_potential_host(mhs_ctx* ctx, void* P_host)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!P_host) return fail(ctx, MHS_ERR_INVALID_ARG, "P is NULL");
    const size_t bytes = (size_t)ctx->L3[0].npts() * ctx->es;
    mhs_status st = ensure_stage(ctx, bytes);
    if (st) return st;
    if ((st = stage_fence(ctx))) return st;
    if ((st = mhs_get_potential(ctx, ctx->stage))) return st;
    CK(cudaMemcpyAsync(P_host, ctx->stage, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return MHS_OK;
}

mhs_status mhs_get_boundary(mhs_ctx* ctx, void* P0)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L2.empty()) return fail(ctx, MHS_ERR_STATE, "context was not created successfully");
    if (!P0) return fail(ctx, MHS_ERR_INVALID_ARG, "P0 is NULL");
    Scope sc(ctx, MHS_KC_PACK);
    launch_unpack(ctx, ctx->L2[0], ctx->L2[0].u, P0);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_get_boundary_host(mhs_ctx* ctx, void* P0_host)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L2.empty()) return fail(ctx, MHS_ERR_STATE, "context was not created successfully");
    if (!P0_host) return fail(ctx, MHS_ERR_INVALID_ARG, "P0 is NULL");
    // (the magnetogram's device copy has been consumed by the solve: it serves as the dense staging plane)
    const size_t bytes = (size_t)ctx->grid.nx * ctx->grid.ny * ctx->es;
    mhs_status st = mhs_get_boundary(ctx, ctx->bz_stage);
    if (st) return st;
    CK(cudaMemcpyAsync(P0_host, ctx->bz_stage, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return MHS_OK;
}

mhs_status mhs_set_potential(mhs_ctx* ctx, const void* P)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!P) return fail(ctx, MHS_ERR_INVALID_ARG, "P is NULL");
    Level& l3 = ctx->L3[0];
    Scope sc(ctx, MHS_KC_PACK);
    launch_pack(ctx, l3, P, l3.u, true, false);
    CK(cudaMemcpyAsync(l3.tmp, l3.u, (size_t)l3.sp * ctx->es, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaGetLastError());
    ctx->have_boundary = true;
    ctx->have_r0 = false;
    ctx->fmg_pending = false;   // (a potential given by the caller is continued from, never replaced)
    return MHS_OK;
}

mhs_status mhs_fields(mhs_ctx* ctx, void* B, void* p, void* rho)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "context was not created successfully");
    if (!ctx->have_boundary) return fail(ctx, MHS_ERR_STATE, "mhs_fields before a successful mhs_solve_boundary / mhs_set_potential");
    if (!B && !p && !rho) return MHS_OK;
    Scope sc(ctx, MHS_KC_FIELDS);
    const Level& l0 = ctx->L3[0];
    if (ctx->wall_ctx) {
        // the nodes next to a side or top wall take the wall values of P through the central differences: the general
        // one-thread-per-node kernel on the dense P = P_h + W
        launch_unpack(ctx, l0, l0.u, ctx->dense_P);
        launch_wall_add(ctx, l0, ctx->wall, ctx->dense_P);
        launch_fields_ref(ctx, l0, ctx->dense_P, B, p, rho, false, true);
        CK(cudaGetLastError());
        return MHS_OK;
    }
    if (!(ctx->opt.flags & (MHS_FLAG_REFERENCE_KERNELS | MHS_FLAG_LOADED_FIELDS)) && launch_fields_ring(ctx, l0, l0.u, B, p, rho)) {
        ctx->prof.ring_fields += 1;
        launch_fields_ref(ctx, l0, l0.u, B, p, rho, true);
    } else if (!(ctx->opt.flags & MHS_FLAG_REFERENCE_KERNELS) && fields_z_ok(ctx, l0)) {
        launch_fields_z(ctx, l0, l0.u, B, p, rho);
        launch_fields_ref(ctx, l0, l0.u, B, p, rho, true);
    } else {
        launch_fields_ref(ctx, l0, l0.u, B, p, rho);
    }
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_diagnostics(mhs_ctx* ctx, const void* B, void* absB, void* J, void* absJ)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!B) return fail(ctx, MHS_ERR_INVALID_ARG, "B is NULL");
    if (ctx->grid.nz < 3) return fail(ctx, MHS_ERR_GRID, "diagnostics need at least 3 planes");
    if (!absB && !J && !absJ) return MHS_OK;
    Scope sc(ctx, MHS_KC_FIELDS);
    launch_diagnostics(ctx, ctx->L3[0], B, absB, J, absJ);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_fieldlines(mhs_ctx* ctx, const void* B, int nseeds, const void* seeds, double step, int max_points, int direction,
                          double bmin, void* lines, int* npoints)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!B || !seeds || !lines || !npoints) return fail(ctx, MHS_ERR_INVALID_ARG, "NULL argument");
    if (nseeds < 0 || !(step > 0.0) || max_points < 1 || !(bmin >= 0.0) || (direction != 1 && direction != -1))
        return fail(ctx, MHS_ERR_INVALID_ARG, "need nseeds >= 0, step > 0, max_points >= 1, bmin >= 0, direction = +1 / -1");
    if (nseeds == 0) return MHS_OK;
    Scope sc(ctx, MHS_KC_FIELDS);
    launch_fieldlines(ctx, ctx->L3[0], B, nseeds, seeds, step, max_points, direction, bmin, lines, npoints);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_fields_host_async(mhs_ctx* ctx, void* B, void* p, void* rho)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->L3.empty()) return fail(ctx, MHS_ERR_STATE, "this context has no 3D grid (nz = 1: boundary solve only)");
    if (!ctx->have_boundary) return fail(ctx, MHS_ERR_STATE, "mhs_fields_host before a successful mhs_solve_boundary / mhs_set_potential");
    const size_t nb = (size_t)ctx->L3[0].npts() * ctx->es;
    mhs_status st = ensure_stage(ctx, 5 * nb);
    if (st) return st;
    if (!ctx->copy_stream) {
        CK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->ev_fields, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->ev_copied, cudaEventDisableTiming));
    }
    if ((st = stage_fence(ctx))) return st;     // the previous results must have left the staging buffer
    char* s = (char*)ctx->stage;
    if ((st = mhs_fields(ctx, B ? s : nullptr, p ? s + 3 * nb : nullptr, rho ? s + 4 * nb : nullptr))) return st;
    CK(cudaEventRecord(ctx->ev_fields, ctx->stream));
    CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_fields, 0));
    if (B) CK(cudaMemcpyAsync(B, s, 3 * nb, cudaMemcpyDeviceToHost, ctx->copy_stream));
    if (p) CK(cudaMemcpyAsync(p, s + 3 * nb, nb, cudaMemcpyDeviceToHost, ctx->copy_stream));
    if (rho) CK(cudaMemcpyAsync(rho, s + 4 * nb, nb, cudaMemcpyDeviceToHost, ctx->copy_stream));
    CK(cudaEventRecord(ctx->ev_copied, ctx->copy_stream));
    ctx->copy_pending = true;
    return MHS_OK;
}

mhs_status mhs_host_sync(mhs_ctx* ctx)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    if (ctx->copy_pending) {
        CK(cudaEventSynchronize(ctx->ev_copied));
        ctx->copy_pending = false;
    }
    drain_events(ctx);
    return MHS_OK;
}

mhs_status mhs_fields_host(mhs_ctx* ctx, void* B, void* p, void* rho)
{
    mhs_status st = mhs_fields_host_async(ctx, B, p, rho);
    if (st) return st;
    return mhs_host_sync(ctx);
}

mhs_status mhs_get_profile(mhs_ctx* ctx, mhs_profile* out)
{
    if (!ctx || !out) return MHS_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(ctx->stream));
    drain_events(ctx);
    *out = ctx->prof;
    return MHS_OK;
}

mhs_status mhs_set_profiling(mhs_ctx* ctx, int level)
{
    if (!ctx || level < 0 || level > 2) return MHS_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(ctx->stream));
    drain_events(ctx);
    ctx->opt.profile = level;
    return MHS_OK;
}

mhs_status mhs_reset_profile(mhs_ctx* ctx)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(ctx->stream));
    drain_events(ctx);
    memset(&ctx->prof, 0, sizeof ctx->prof);
    return MHS_OK;
}

// ---- operator-level access ------------------------------------------------------------------
int mhs_num_levels(const mhs_ctx* ctx, int dim)
{
    if (!ctx) return 0;
    return dim == 3 ? (int)ctx->L3.size() : dim == 2 ? (int)ctx->L2.size() : 0;
}

mhs_status mhs_level_dims(const mhs_ctx* cctx, int dim, int level, int* nx, int* ny, int* nz)
{
    mhs_ctx* ctx = const_cast<mhs_ctx*>(cctx);
    if (!ctx) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    if (nx) *nx = (*Ls)[level].nx;
    if (ny) *ny = (*Ls)[level].ny;
    if (nz) *nz = (*Ls)[level].nz;
    return MHS_OK;
}

static void* pick(Level& lv, int which) { return which == 0 ? lv.u : which == 1 ? lv.rhs : which == 2 ? lv.r : nullptr; }

mhs_status mhs_level_set(mhs_ctx* ctx, int dim, int level, int which, const void* src)
{
    if (!ctx || !src) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    Level& lv = (*Ls)[level];
    void* dst = pick(lv, which);
    if (!dst) return fail(ctx, MHS_ERR_INVALID_ARG, "this level has no such array");
    Scope sc(ctx, MHS_KC_PACK);
    const bool bottom = dim == 3 && level == 0 && which == 0;
    launch_pack(ctx, lv, src, dst, bottom, false);
    if (bottom) {
        CK(cudaMemcpyAsync(lv.tmp, lv.u, (size_t)lv.sp * ctx->es, cudaMemcpyDeviceToDevice, ctx->stream));
        ctx->have_r0 = false;
        ctx->fmg_pending = false;
        ctx->have_boundary = true;   // (the same as mhs_set_potential)
    }
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_level_get(mhs_ctx* ctx, int dim, int level, int which, void* dst)
{
    if (!ctx || !dst) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    Level& lv = (*Ls)[level];
    void* src = pick(lv, which);
    if (!src) return fail(ctx, MHS_ERR_INVALID_ARG, "this level has no such array");
    Scope sc(ctx, MHS_KC_PACK);
    launch_unpack(ctx, lv, src, dst);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_smooth(mhs_ctx* ctx, int dim, int level, int sweeps)
{
    if (!ctx || sweeps < 0) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    if ((*Ls)[level].coarsest) return fail(ctx, MHS_ERR_INVALID_ARG, "the coarsest level is solved exactly, not smoothed");
    smooth(ctx, *Ls, level, sweeps, nullptr);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_residual(mhs_ctx* ctx, int dim, int level)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    Level& lv = (*Ls)[level];
    if (!lv.r) return fail(ctx, MHS_ERR_INVALID_ARG, "the coarsest level has no residual array");
    Scope sc(ctx, kc_for(lv, level, 1));
    launch_residual_ref(ctx, lv, lv.u, lv.rhs, lv.r, nullptr);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_restrict(mhs_ctx* ctx, int dim, int level)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    Level& lv = (*Ls)[level];
    if (lv.coarsest) return fail(ctx, MHS_ERR_INVALID_ARG, "no level below the coarsest");
    Scope sc(ctx, kc_for(lv, level, 1));
    const void* rhs = lv.rhs;
    if (use_fast(ctx, lv)) {
        restrict_fast(ctx, lv, lv.u, rhs, (*Ls)[level + 1], 0, nullptr);
    } else {
        launch_residual_ref(ctx, lv, lv.u, rhs, lv.r, nullptr);
        launch_restrict_ref(ctx, lv, lv.r, (*Ls)[level + 1], (*Ls)[level + 1].rhs, nullptr);
    }
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_prolong(mhs_ctx* ctx, int dim, int level)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    Level& lv = (*Ls)[level];
    if (lv.coarsest) return fail(ctx, MHS_ERR_INVALID_ARG, "no level below the coarsest");
    Scope sc(ctx, kc_for(lv, level, 2));
    if (use_fast(ctx, lv)) launch_prolong_v(ctx, lv, lv.u, (*Ls)[level + 1], (*Ls)[level + 1].u, 0, nullptr);
    else launch_prolong_ref(ctx, lv, lv.u, (*Ls)[level + 1], (*Ls)[level + 1].u, nullptr);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_vcycle(mhs_ctx* ctx, int dim, int level)
{
    if (!ctx) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    vcycle(ctx, *Ls, level, nullptr);
    CK(cudaGetLastError());
    return MHS_OK;
}

mhs_status mhs_op_resnorm(mhs_ctx* ctx, int dim, int level, double* out_host)
{
    if (!ctx || !out_host) return MHS_ERR_INVALID_ARG;
    std::vector<Level>* Ls;
    mhs_status st = check_level(ctx, dim, level, &Ls);
    if (st) return st;
    {
        const long long np = resnorm_partials(ctx, *Ls, level, nullptr);
        norm_final(ctx, (*Ls)[level], level, np, 2);
    }
    { mhs_status rs = read_ctl(ctx); if (rs) return rs; }
    drain_events(ctx);
    *out_host = ctx->ctl_host->r_last;
    return MHS_OK;
}

}  // extern "C"
