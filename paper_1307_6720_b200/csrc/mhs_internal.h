// Internal declarations of libmhs_b200 (not part of the ABI; see include/mhs.h).
//
// Device layout of one level ("aliased Dirichlet" layout):
//   a level with nx x ny x nz vertices is stored with row pitch sx = nx-1 and sy = ny-1 rows per
//   plane, node (i,j,k) at  base[i + sx*(j + sy*k)].  The Dirichlet-zero node (nx-1, j, k) IS node
//   (0, j+1, k), and row (., ny-1, k) IS row (., 0, k+1): every wall value exists once, is zero, and
//   is never written, so rows are 2^m elements long (128-byte aligned for the big levels), no
//   padding bytes are streamed, and stencil reads at i+-1 / j+-1 never need a bounds test.
//   One zero plane in front of k = 0 and one behind k = nz-1 (+ a row) absorb the remaining
//   out-of-range neighbour reads.  2D levels are the same with nz = 1.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <string>
#include <vector>

#include "mhs.h"

namespace mhs {

// Per-level parameters handed to kernels by value.
template <typename T>
struct LP {
    int nx, ny, nz;   // vertices (nz = 1 in 2D)
    int sx, sy;       // row pitch, rows per plane
    long long sp;     // plane stride = sx*sy
    const T* tab;     // device: cx[nz] | cy[nz] | diag[nz] | w[nz]   (cx = c_k/hx^2, w = omega/diag)
    T cz, a2;         // 1/hz^2 (0 in 2D), alpha^2 (0 in 2D)
};

struct Ctl {  // device-side solve control block (one per context)
    int done;        // 1: stop rule met -> every later cycle kernel returns at once
    int cycles;      // cycles completed in this call
    int max_cycles;
    int nan_seen;
    int stag_on, stag_count, stagnated;
    int units;       // cycles completed so far (device-side counter of the unit scheme)  // fp32 stagnation rule (C20)
    double r0, tol, r_last;
    double hist[MHS_HISTORY_LEN];
};

struct Level {
    int dim = 3;
    int nx = 0, ny = 0, nz = 1, sx = 0, sy = 0;
    long long sp = 0, pad = 0, alloc = 0;
    double hx = 0, hy = 0, hz = 0;
    bool coarsest = false;
    void *u = nullptr, *tmp = nullptr, *rhs = nullptr, *r = nullptr;  // -> node (0,0,0)
    void *raw[4] = {nullptr, nullptr, nullptr, nullptr};
    void* tab = nullptr;
    std::vector<double> c;  // 1 + f at this level's planes
    int ncoarse = 0;        // unknowns of the exact solve (coarsest level only)
    void* ainv = nullptr;   // device T[ncoarse^2]
    void* zl = nullptr;     // device T[2*nz]: Thomas factors cp | 1/den of the z-line smoother (mhs_options.smoother = 1)
    long long npts() const { return (long long)nx * ny * nz; }
};

struct Ev { int kc; cudaEvent_t a, b; };

}  // namespace mhs

struct mhs_ctx {
    mhs_grid grid{};
    mhs_options opt{};
    double alpha = 0;
    int es = 8;  // element size
    cudaStream_t stream = nullptr;
    std::vector<mhs::Level> L3, L2;
    std::vector<double> f, dfdz, p_b, rho_b;
    void* prof_tab = nullptr;  // device T[4*nz]: xi | dxi | p_b | rho_b
    mhs::Ctl* ctl = nullptr;   // device
    mhs::Ctl* ctl_host = nullptr;  // pinned
    double* partial = nullptr;     // device partial sums of the norm
    long long npartial = 0;
    void* stage = nullptr;         // device staging for host-pointer entry points (lazy)
    size_t stage_bytes = 0;
    void* bz_stage = nullptr;      // device copy of a host magnetogram (mhs_solve_boundary_host)
    cudaStream_t copy_stream = nullptr;                  // device -> host copies of mhs_fields_host_async
    cudaEvent_t ev_fields = nullptr, ev_copied = nullptr;
    bool copy_pending = false;
    bool have_boundary = false, have_r0 = false;
    // Dirichlet data on the side / top faces (mhs_bc = MHS_BC_DIRICHLET_DATA; mhs_kernels_wall.cu): W = the data on the wall nodes,
    // zero elsewhere (dense, N elements); the finest level then has a right-hand side (-L W); dense_P: N elements of scratch
    bool wall_ctx = false;
    int bc_sides = 0, bc_top = 0;
    void *wall = nullptr, *dense_P = nullptr;
    bool fmg_pending = false;          // mhs_solve_boundary has run and no interior cycle yet: the FMG start may replace the interior
    const mhs::Level* ref_level = nullptr;   // a level that must run the general reference kernels right now (FMG start)
    double r0_interior = 0;
    mhs_profile prof{};
    int cur_kc = MHS_KC_PACK;  // kernel class the launchers charge
    int num_sms = 148;
    int device = 0;            // the CUDA device the context was created on
    bool debug = false;        // MHS_DEBUG was set at create: launch shapes go to stderr
    bool no_align = false;     // MHS_NO_ALIGN was set at create: k_zsweep keeps the cost-balanced ranges (A/B of the aligned z-segments)
    long long cl3_pts = 0;     // levels of a big 3D hierarchy up to this many nodes run inside the cluster kernel (cluster_start(); knob MHS_CL3_PTS)
    long long rb_pts = 40000;   // levels up to this many nodes restrict with the box kernel (k_resid_restrict_box; knob MHS_RB_PTS, 0 = off)
    long long s2_pts = 40000;   // levels up to this many nodes (33^3) smooth two sweeps per launch (k_smooth2_node; knob MHS_S2_PTS, 0 = off; measured at 257^3: off 3235, 40000: 3255, 300000: 3250 V-cycles/s)
    long long mid_pts = 5000000;   // levels up to this many nodes are 'mid levels' (mid_level(); tuning knob MHS_MID_PTS, read at create)
    int tail3 = 1 << 30, tail2 = 1 << 30;  // first level kept in shared memory by the cluster kernel's CTA 0
    int clus3 = 1 << 30, clus2 = 1 << 30;  // first level handled by the cluster kernel (<= tail; mhs_kernels_cluster.cu)
    int cluster_max = 8;                   // largest thread-block cluster the device co-schedules (<= 16)
    int dir = 0;               // z traversal direction of the next big kernel (alternates)
    long long pending_norm = 0;   // partial sums of a norm whose stop rule the next finest-level restriction is to apply (vcycle)
    std::vector<mhs::Ev> ev_pending;
    std::vector<cudaEvent_t> ev_pool;
    std::string err;
};

namespace mhs {

inline void count_launch(mhs_ctx* c) { c->prof.launches[c->cur_kc] += 1; }

// One-time per-kernel setup (cudaFuncSetAttribute applies to the CURRENT device only) and cached occupancy figures are
// kept per device: a second context on another GPU of the same process must get its own.  `fn` returns a non-zero int
// (the cached value); concurrent first calls may both run it -- it is idempotent.
constexpr int MAX_DEVICES = 64;
struct PerDevice {
    std::atomic<int> v[MAX_DEVICES];
    PerDevice() { for (auto& a : v) a.store(0, std::memory_order_relaxed); }
};
template <typename F>
inline int per_device(PerDevice& pd, const mhs_ctx* c, F fn)
{
    const int d = c->device >= 0 && c->device < MAX_DEVICES ? c->device : 0;
    int x = pd.v[d].load(std::memory_order_acquire);
    if (!x) {
        x = fn();
        pd.v[d].store(x, std::memory_order_release);
    }
    return x;
}

// Kernels that live on the L1 (no dynamic shared memory) say so ONCE: with no stated preference a kernel launched after one
// that had the SM configured for 220 KB of shared memory (k_zsweep, the cluster kernel's tail) inherits that split and runs
// with a ~28 KB L1 -- measured: residual+restriction 44 -> 61 us, 25 us per zsweep/restriction pair.
template <typename K>
inline void prefer_l1(K kern)
{
    cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxL1);
}

// Launch with the programmatic-stream-serialization attribute (PDL, see pdl_enter() in mhs_device.cuh).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(const mhs_ctx* c, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = (c->opt.flags & MHS_FLAG_NO_PDL) ? 0 : 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ---- launchers of the reference kernels (mhs_kernels_ref.cu) --------------------------------
// `done` (may be NULL) points at Ctl::done: when set, the kernel returns without doing anything.
void launch_smooth_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done);
void launch_residual_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* r, const int* done);
void launch_restrict_ref(mhs_ctx* c, const Level& fine, const void* r, const Level& coarse, void* rhs_c, const int* done);
void launch_prolong_ref(mhs_ctx* c, const Level& fine, void* u, const Level& coarse, const void* ec, const int* done);
void launch_coarse_solve(mhs_ctx* c, const Level& lv, void* u, const void* rhs, const int* done);
// partial sums of (rhs - L u)^2 -> c->partial[0..n); returns n
long long launch_resnorm_partial_ref(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, const int* done);
long long resnorm_partial_capacity(const Level& lv);
// mode 0: r0 = norm; mode 1: record a cycle (history, stop rule); mode 2: r_last only
void launch_norm_final(mhs_ctx* c, long long n, int mode);
void launch_pack(mhs_ctx* c, const Level& lv, const void* dense, void* dst, bool keep_bottom, bool negate);
void launch_unpack(mhs_ctx* c, const Level& lv, const void* src, void* dense);
// dense: P is a dense array (pitch nx, walls stored) instead of the level's aliased layout
void launch_fields_ref(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho, bool ends_only = false, bool dense = false);
// ---- Dirichlet data on the side / top faces (mhs_kernels_wall.cu) ----
void launch_wall_take(mhs_ctx* c, const Level& lv, int sides, int top, const void* G, void* W);
void launch_wall_rhs(mhs_ctx* c, const Level& lv, const void* W, void* rhs);
void launch_wall_add(mhs_ctx* c, const Level& lv, const void* W, void* P);
// ---- one-pass field recovery (mhs_kernels_fields.cu): planes 1 .. nz-2 ----
bool fields_z_ok(const mhs_ctx* c, const Level& lv);
void launch_fields_z(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho);
// the same, fed by the bulk-copy engine (mhs_kernels_fields_ring.cu); false: shape not supported, nothing launched
bool launch_fields_ring(mhs_ctx* c, const Level& lv, const void* P, void* B, void* p, void* rho);
void launch_diagnostics(mhs_ctx* c, const Level& lv, const void* B, void* absB, void* J, void* absJ);
// ---- solver variants (mhs_kernels_variants.cu): z-line Jacobi, full-multigrid start ----
bool zline_ok(const mhs_ctx* c, const Level& lv);
void launch_zline(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done);
void launch_inject_bottom(mhs_ctx* c, const Level& fine, const void* fine_u, const Level& lv, int stride, void* a, void* b);
void launch_bottom_rhs(mhs_ctx* c, const Level& lv, const void* u, void* rhs);
// ---- field-line integration (mhs_kernels_lines.cu) ----
void launch_fieldlines(mhs_ctx* c, const Level& lv, const void* B, int nseeds, const void* seeds, double step, int max_points, int direction,
                       double bmin, void* lines, int* npoints);

// ---- tuned 3D kernels (mhs_kernels_fast.cu) ----
bool fast_ok(const mhs_ctx* c, const Level& lv);
bool mid_level(const mhs_ctx* c, const Level& lv);   // small enough to live in the L2: parallelism-bound, gets fine-grained launch shapes
// mode 0: sweep; 1: sweep + partial sums of the INPUT's ||rhs - L u||^2; 2: partial sums only; 3: the first two sweeps
// from the zero initial guess in one pass (u not read).  Returns #partials.
long long launch_smooth_z(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int mode, int reverse, const int* done);
long long smooth_z_partial_capacity(const mhs_ctx* c, const Level& lv);
void launch_scale_rhs(mhs_ctx* c, const Level& lv, const void* rhs, void* u, const int* done);
// residual + full weighting as a box kernel (levels up to c->rb_pts nodes with a right-hand side)
bool resid_restrict_box_ok(const mhs_ctx* c, const Level& fine);
void launch_resid_restrict_box(mhs_ctx* c, const Level& fine, const void* u, const void* rhs, const Level& coarse, void* rhs_c, const int* done);
// two sweeps in one launch, one thread per node (levels up to c->s2_pts nodes with a right-hand side)
bool smooth2_node_ok(const mhs_ctx* c, const Level& lv);
void launch_smooth2_node(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, const int* done);
void launch_resid_restrict_z(mhs_ctx* c, const Level& fine, const void* u, const void* rhs, const Level& coarse, void* rhs_c, int reverse, const int* done);
// the same for a big level, in separable form (no plane of u kept, the residual never formed)
void launch_resid_restrict_sep(mhs_ctx* c, const Level& fine, const void* u, const void* rhs, const Level& coarse, void* rhs_c, int reverse, const int* done);
// the same for a level WITHOUT a right-hand side (the finest 3D level), fed by the bulk-copy engine (mhs_kernels_restrict.cu);
// down: walk down in z.  false: shape not supported, nothing launched.
// norm_n > 0: the cycle's stop rule (the reduction of c->partial[0 .. norm_n) and stop_rule, i.e. k_norm_final mode 1) is done by
// CTA 0 of this kernel before its own work; false then also means "not folded in, nothing launched".
bool launch_resid_restrict_ring(mhs_ctx* c, const Level& fine, const void* u, const Level& coarse, void* rhs_c, int down, const int* done,
                                long long norm_n = 0);
void launch_prolong_v(mhs_ctx* c, const Level& fine, void* u, const Level& coarse, const void* ec, int reverse, const int* done);
// ---- temporally blocked smoother (mhs_kernels_zfused.cu) ----
bool zsweep_ok(const mhs_ctx* c, const Level& lv);
// S (1 or 2) sweeps in one pass, u -> out.  zero: u is identically zero and not read.  norm: partial sums of the
// squared residual of u go to c->partial; returns their number.
int launch_zsweep(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int S, bool zero, bool norm, const int* done);

// the same applied to u + P e_c (prolongation + correction folded into the pass; u is not modified).  false: not launched
// (the level cannot run in k_zsweep) -- the caller prolongs separately.
bool launch_zsweep_prolong(mhs_ctx* c, const Level& lv, const void* u, const void* rhs, void* out, int S, const Level& coarse, const void* ec,
                           const int* done);

// ---- the small-level cluster kernel (mhs_kernels_cluster.cu) ----
int tail_start(const mhs_ctx* c, const std::vector<Level>& Ls, size_t budget_bytes);
int cluster_start(const mhs_ctx* c, const std::vector<Level>& Ls, int tail);
int cluster_max_size(const mhs_ctx* c);
// mode 0: V pass from level lc >= 1 with zero initial guess; 1: one V-cycle continuing from level 0 (lc == 0);
// 2: the whole solve loop on level 0 (norm, stop rule in c->ctl, V-cycle) in one launch.
void launch_cluster(mhs_ctx* c, std::vector<Level>& Ls, int lc, int mode, const int* done);

}  // namespace mhs
