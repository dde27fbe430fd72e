"""Thin Python binding of the C-ABI library libmhs_b200.so (include/mhs.h): argument marshalling
only.  PyTorch supplies device memory and streams; every step of the path runs in the library's
CUDA kernels.  There is NO CPU fallback: if the library cannot be built/loaded, or no CUDA device is
present, the calls raise.

Module-level functions carry the C names (mhs_create, mhs_solve_boundary, mhs_solve_interior,
mhs_fields, mhs_destroy, ...); `Solver` is a small convenience wrapper over them.
Arrays are torch tensors shaped (nz, ny, nx) / (ny, nx): x fastest, as the ABI wants.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

MHS_F32, MHS_F64 = 0, 1
MHS_FLAG_REFERENCE_KERNELS = 1
MHS_FLAG_SYNC_EACH_CYCLE = 2
MHS_FLAG_UNFUSED_KERNELS = 4
MHS_FLAG_BIG_LEVEL_KERNELS = 8
MHS_FLAG_SEPARATE_PROLONG = 16
MHS_FLAG_NO_PDL = 32
MHS_FLAG_LOADED_RESTRICT = 64
MHS_FLAG_LOADED_FIELDS = 128
MHS_FLAG_NO_FOLDED_NORM = 256
MHS_SMOOTH_JACOBI, MHS_SMOOTH_ZLINE = 0, 1
MHS_HISTORY_LEN = 256
MHS_KC_COUNT = 8
(MHS_OK, MHS_ERR_INVALID_ARG, MHS_ERR_GRID, MHS_ERR_NOT_ELLIPTIC, MHS_ERR_INDEFINITE, MHS_ERR_STATE,
 MHS_ERR_NOT_CONVERGED, MHS_ERR_CUDA, MHS_ERR_OOM) = range(9)

EXPORTS = [
    "mhs_default_options", "mhs_create", "mhs_destroy", "mhs_solve_boundary", "mhs_solve_boundary_host",
    "mhs_solve_interior", "mhs_solve_batch", "mhs_fields", "mhs_fields_host", "mhs_fields_host_async", "mhs_host_sync", "mhs_diagnostics", "mhs_fieldlines", "mhs_get_potential", "mhs_get_potential_host",
    "mhs_set_potential", "mhs_get_boundary", "mhs_get_boundary_host", "mhs_last_error", "mhs_status_string", "mhs_get_profile", "mhs_reset_profile",
    "mhs_kernel_class_name", "mhs_set_profiling", "mhs_num_levels", "mhs_level_dims", "mhs_level_set", "mhs_level_get",
    "mhs_op_smooth", "mhs_op_residual", "mhs_op_restrict", "mhs_op_prolong", "mhs_op_vcycle", "mhs_op_resnorm",
    "mhs_resnorm_static", "mhs_static_last_error", "mhs_set_wall_data",
]
MHS_BC_DIRICHLET_ZERO, MHS_BC_DIRICHLET_DATA = 0, 1
MHS_STATIC_SCRATCH_DOUBLES = 65536


class mhs_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("Lx", C.c_double), ("Ly", C.c_double), ("Lz", C.c_double)]


class mhs_bc(C.Structure):
    _fields_ = [("sides", C.c_int), ("top", C.c_int)]


class mhs_options(C.Structure):
    _fields_ = [("dtype", C.c_int), ("omega", C.c_double), ("n_pre", C.c_int), ("n_post", C.c_int),
                ("max_levels", C.c_int), ("boundary_tol", C.c_double), ("boundary_max_cycles", C.c_int),
                ("mu0", C.c_double), ("g", C.c_double),
                ("p_b", C.POINTER(C.c_double)), ("rho_b", C.POINTER(C.c_double)), ("dfdz", C.POINTER(C.c_double)),
                ("stream", C.c_void_p), ("profile", C.c_int), ("flags", C.c_int), ("smoother", C.c_int), ("fmg_cycles", C.c_int)]


class mhs_solve_info(C.Structure):
    _fields_ = [("cycles", C.c_int), ("r0", C.c_double), ("r_final", C.c_double),
                ("history", C.c_double * MHS_HISTORY_LEN), ("stagnated", C.c_int)]


class mhs_profile(C.Structure):
    _fields_ = [("launches", C.c_longlong * MHS_KC_COUNT), ("ms", C.c_double * MHS_KC_COUNT),
                ("sweeps_l0", C.c_longlong), ("fused_prolong_l0", C.c_longlong), ("xtiled_zsweep", C.c_longlong),
                ("ring_restrict", C.c_longlong), ("ring_fields", C.c_longlong)]


class MHSError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (status_string(status), msg))
        self.status = status


_lib = None


def lib():
    """Load (building first if the in-tree .so is missing or stale) libmhs_b200.so.  Raises if that
    is impossible -- the product has no other code path."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if os.environ.get("MHS_NO_BUILD") != "1":
            path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libmhs_b200.so is missing (python -m paper_1307_6720_b200.build); no CPU fallback exists")
        L = C.CDLL(path)
        vp, ip, dp = C.c_void_p, C.c_int, C.c_double
        L.mhs_default_options.argtypes = [C.POINTER(mhs_options)]
        L.mhs_default_options.restype = None
        L.mhs_create.argtypes = [C.POINTER(mhs_grid), dp, C.POINTER(C.c_double), C.POINTER(mhs_bc),
                                 C.POINTER(mhs_options), C.POINTER(vp)]
        L.mhs_destroy.argtypes = [vp]
        L.mhs_destroy.restype = None
        for n in ("mhs_solve_boundary", "mhs_solve_boundary_host"):
            getattr(L, n).argtypes = [vp, vp, C.POINTER(mhs_solve_info)]
        L.mhs_solve_interior.argtypes = [vp, dp, ip, C.POINTER(mhs_solve_info)]
        L.mhs_solve_batch.argtypes = [vp, ip, vp, dp, ip, vp, vp, vp, vp, C.POINTER(mhs_solve_info)]
        for n in ("mhs_fields", "mhs_fields_host", "mhs_fields_host_async"):
            getattr(L, n).argtypes = [vp, vp, vp, vp]
        L.mhs_host_sync.argtypes = [vp]
        L.mhs_diagnostics.argtypes = [vp, vp, vp, vp, vp]
        L.mhs_fieldlines.argtypes = [vp, vp, ip, vp, dp, ip, ip, dp, vp, vp]
        for n in ("mhs_get_potential", "mhs_get_potential_host", "mhs_set_potential", "mhs_get_boundary", "mhs_get_boundary_host", "mhs_set_wall_data"):
            getattr(L, n).argtypes = [vp, vp]
        L.mhs_last_error.argtypes = [vp]
        L.mhs_last_error.restype = C.c_char_p
        L.mhs_status_string.argtypes = [ip]
        L.mhs_status_string.restype = C.c_char_p
        L.mhs_get_profile.argtypes = [vp, C.POINTER(mhs_profile)]
        L.mhs_reset_profile.argtypes = [vp]
        L.mhs_set_profiling.argtypes = [vp, ip]
        L.mhs_kernel_class_name.argtypes = [ip]
        L.mhs_kernel_class_name.restype = C.c_char_p
        L.mhs_num_levels.argtypes = [vp, ip]
        L.mhs_level_dims.argtypes = [vp, ip, ip, C.POINTER(ip), C.POINTER(ip), C.POINTER(ip)]
        L.mhs_level_set.argtypes = [vp, ip, ip, ip, vp]
        L.mhs_level_get.argtypes = [vp, ip, ip, ip, vp]
        L.mhs_op_smooth.argtypes = [vp, ip, ip, ip]
        for n in ("mhs_op_residual", "mhs_op_restrict", "mhs_op_prolong", "mhs_op_vcycle"):
            getattr(L, n).argtypes = [vp, ip, ip]
        L.mhs_op_resnorm.argtypes = [vp, ip, ip, C.POINTER(C.c_double)]
        L.mhs_resnorm_static.argtypes = [vp, ip, ip, ip, ip, dp, dp, dp, dp, vp, vp, vp]
        L.mhs_static_last_error.argtypes = []
        L.mhs_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def status_string(s) -> str:
    return lib().mhs_status_string(int(s)).decode()


def _check(h, st, allow=()):
    if st != MHS_OK and st not in allow:
        raise MHSError(st, lib().mhs_last_error(h).decode() if h else "")
    return st


def _dptr(t, dtype, numel, device="cuda"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor):
        raise TypeError("expected a torch tensor")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise ValueError("tensor must be contiguous %s with %d elements (got %s, %d)" % (dtype, numel, t.dtype, t.numel()))
    if device == "cuda" and not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if device == "cpu" and t.is_cuda:
        raise ValueError("expected a host tensor")
    return C.c_void_p(t.data_ptr())


def _hd(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _info(i: mhs_solve_info, status):
    n = min(i.cycles, MHS_HISTORY_LEN)
    return dict(cycles=i.cycles, r0=i.r0, r_final=i.r_final, history=np.array(i.history[:n]),
                converged=status == MHS_OK, status=status,
                stagnated=bool(i.stagnated))


# ------------------------------------------------------------------ C-named functions ---------
def mhs_create(nx, ny, nz, Lx, Ly, Lz, alpha, f_profile=None, *, dtype=torch.float64, omega=2.0 / 3.0,
               n_pre=2, n_post=2, max_levels=0, boundary_tol=1e-10, boundary_max_cycles=100, mu0=0.5, g=1.0,
               p_b=None, rho_b=None, dfdz=None, stream=None, profile=0, flags=0, smoother=0, fmg_cycles=0, bc=None):
    """-> opaque context handle (int).  See include/mhs.h: mhs_create.  bc: None or (sides, top) of MHS_BC_*."""
    L = lib()
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: paper_1307_6720_b200 has no CPU fallback")
    torch.cuda.init()
    torch.zeros(1, device="cuda")  # make sure the primary context exists and is current
    o = mhs_options()
    L.mhs_default_options(C.byref(o))
    o.dtype = MHS_F64 if dtype == torch.float64 else MHS_F32
    o.omega, o.n_pre, o.n_post, o.max_levels = omega, n_pre, n_post, max_levels
    o.boundary_tol, o.boundary_max_cycles, o.mu0, o.g = boundary_tol, boundary_max_cycles, mu0, g
    keep = [_hd(p_b), _hd(rho_b), _hd(dfdz), _hd(f_profile)]
    for a in keep:
        if a is not None and a.size != nz:
            raise ValueError("profiles must have nz entries")
    pd = C.POINTER(C.c_double)
    o.p_b = keep[0].ctypes.data_as(pd) if keep[0] is not None else None
    o.rho_b = keep[1].ctypes.data_as(pd) if keep[1] is not None else None
    o.dfdz = keep[2].ctypes.data_as(pd) if keep[2] is not None else None
    s = stream if stream is not None else torch.cuda.current_stream()
    o.stream = C.c_void_p(s.cuda_stream if hasattr(s, "cuda_stream") else int(s))
    o.profile, o.flags = profile, flags
    o.smoother, o.fmg_cycles = smoother, fmg_cycles
    grid = mhs_grid(nx, ny, nz, Lx, Ly, Lz)
    h = C.c_void_p()
    bcs = mhs_bc(int(bc[0]), int(bc[1])) if bc is not None else None
    st = L.mhs_create(C.byref(grid), alpha, keep[3].ctypes.data_as(pd) if keep[3] is not None else None,
                      C.byref(bcs) if bcs is not None else None, C.byref(o), C.byref(h))
    if st != MHS_OK:
        msg = L.mhs_last_error(h).decode() if h else ""
        if h:
            L.mhs_destroy(h)
        raise MHSError(st, msg)
    return h


def mhs_destroy(h):
    if h:
        lib().mhs_destroy(h)


def mhs_solve_boundary(h, Bz0, dtype, nx, ny):
    i = mhs_solve_info()
    if Bz0.is_cuda:
        st = lib().mhs_solve_boundary(h, _dptr(Bz0, dtype, nx * ny), C.byref(i))
    else:
        st = lib().mhs_solve_boundary_host(h, _dptr(Bz0, dtype, nx * ny, "cpu"), C.byref(i))
    _check(h, st, (MHS_ERR_NOT_CONVERGED,))
    return _info(i, st)


def mhs_solve_interior(h, tol, max_cycles):
    i = mhs_solve_info()
    st = lib().mhs_solve_interior(h, tol, max_cycles, C.byref(i))
    _check(h, st, (MHS_ERR_NOT_CONVERGED,))
    return _info(i, st)


def mhs_host_sync(h):
    _check(h, lib().mhs_host_sync(h))


def mhs_fields(h, B, p, rho, dtype, N, host=False, wait=True):
    dev = "cpu" if host else "cuda"
    fn = (lib().mhs_fields_host if wait else lib().mhs_fields_host_async) if host else lib().mhs_fields
    _check(h, fn(h, _dptr(B, dtype, 3 * N, dev), _dptr(p, dtype, N, dev), _dptr(rho, dtype, N, dev)))


def mhs_get_potential(h, P, dtype, N):
    if P.is_cuda:
        _check(h, lib().mhs_get_potential(h, _dptr(P, dtype, N)))
    else:
        _check(h, lib().mhs_get_potential_host(h, _dptr(P, dtype, N, "cpu")))


def mhs_set_potential(h, P, dtype, N):
    _check(h, lib().mhs_set_potential(h, _dptr(P, dtype, N)))


def mhs_resnorm_static(P, c, out, nx, ny, nz, hx, hy, hz, alpha, stream=None):
    """mhs_resnorm_static (include/mhs.h): ||L P||_2 of the dense device tensor P into the 1-element fp64 device tensor
    `out`; c: nz fp64 device values 1 + f(z_k).  Allocates nothing; asynchronous on `stream` (default: torch's current)."""
    if P.dtype not in (torch.float32, torch.float64):
        raise TypeError("P must be float32 or float64")
    s = torch.cuda.current_stream().cuda_stream if stream is None else stream
    st = lib().mhs_resnorm_static(_dptr(P, P.dtype, nx * ny * nz), MHS_F64 if P.dtype == torch.float64 else MHS_F32, nx, ny, nz,
                                  hx, hy, hz, alpha, _dptr(c, torch.float64, nz), _dptr(out, torch.float64, 1), C.c_void_p(s))
    if st != MHS_OK:
        raise MHSError(st, lib().mhs_static_last_error().decode())


def mhs_set_wall_data(h, G, dtype, N):
    _check(h, lib().mhs_set_wall_data(h, _dptr(G, dtype, N)))


def mhs_get_profile(h):
    p = mhs_profile()
    _check(h, lib().mhs_get_profile(h, C.byref(p)))
    names = [lib().mhs_kernel_class_name(k).decode() for k in range(MHS_KC_COUNT)]
    return dict(launches={n: int(p.launches[k]) for k, n in enumerate(names)},
                ms={n: float(p.ms[k]) for k, n in enumerate(names)}, sweeps_l0=int(p.sweeps_l0),
                fused_prolong_l0=int(p.fused_prolong_l0), xtiled_zsweep=int(p.xtiled_zsweep), ring_restrict=int(p.ring_restrict), ring_fields=int(p.ring_fields),
                total_launches=int(sum(p.launches)))


def mhs_reset_profile(h):
    _check(h, lib().mhs_reset_profile(h))


# ------------------------------------------------------------------ convenience wrapper -------
class Solver:
    """One grid + stream.  Mirrors the state machine of include/mhs.h:
    create -> solve_boundary -> solve_interior (repeatable, continues) -> fields."""

    def __init__(self, nx, ny, nz, L=(1.0, 1.0, 1.0), alpha=0.0, f=None, dtype=torch.float64, **opts):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.dtype = dtype
        self.N = self.nx * self.ny * self.nz
        self.h = mhs_create(self.nx, self.ny, self.nz, L[0], L[1], L[2], alpha, f, dtype=dtype, **opts)

    @classmethod
    def from_workload(cls, w, **over):
        dt = torch.float64 if w.dtype == "f64" else torch.float32
        kw = dict(omega=w.omega, n_pre=w.n_pre, n_post=w.n_post, mu0=w.mu0, g=w.g, p_b=w.p_b, rho_b=w.rho_b,
                  boundary_tol=w.tol)
        kw.update(over)
        return cls(w.nx, w.ny, w.nz, w.L, w.alpha, w.f, dtype=kw.pop("dtype", dt), **kw)

    def close(self):
        h, self.h = getattr(self, "h", None), None
        if h and _lib is not None:      # (at interpreter exit the module may already be torn down)
            _lib.mhs_destroy(h)         # (synchronises the copy stream before anything is freed)
        self._inflight = []

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the five calls of the north star
    def solve_boundary(self, Bz0):
        return mhs_solve_boundary(self.h, Bz0, self.dtype, self.nx, self.ny)

    def solve_interior(self, tol=1e-10, max_cycles=100):
        return mhs_solve_interior(self.h, tol, max_cycles)

    def solve_batch(self, Bz0, tol=1e-10, max_cycles=100, want=("P",)):
        """mhs_solve_batch: Bz0 (nb, ny, nx) device tensor -> dict of outputs ("P" (nb, nz, ny, nx), "B" (nb, 3, nz, ny, nx),
        "p", "rho") and the list of per-member interior-solve infos."""
        nb = int(Bz0.shape[0])
        shp = (self.nz, self.ny, self.nx)
        mk = lambda *s: torch.empty(s, dtype=self.dtype, device="cuda")
        out = {k: (mk(nb, 3, *shp) if k == "B" else mk(nb, *shp)) for k in want}
        infos = (mhs_solve_info * max(nb, 1))()
        ptr = lambda k, m: _dptr(out[k].reshape(-1), self.dtype, nb * m) if k in out else None
        st = lib().mhs_solve_batch(self.h, nb, _dptr(Bz0.reshape(-1), self.dtype, nb * self.nx * self.ny), tol, max_cycles,
                                   ptr("P", self.N), ptr("B", 3 * self.N), ptr("p", self.N), ptr("rho", self.N), infos)
        _check(self.h, st, (MHS_ERR_NOT_CONVERGED,))
        # (a member's own status: converged unless it used up max_cycles above the tolerance)
        res = []
        for b in range(nb):
            i = infos[b]
            ok = i.r_final <= tol * i.r0 or bool(i.stagnated)
            res.append(_info(i, MHS_OK if ok else MHS_ERR_NOT_CONVERGED))
        return out, res

    def host_sync(self):
        mhs_host_sync(self.h)
        self._inflight = []

    def fields(self, B=None, p=None, rho=None, want=("B", "p", "rho"), host=False, wait=True):
        dev = "cpu" if host else "cuda"
        mk = lambda n: torch.empty(n, dtype=self.dtype, device=dev, pin_memory=host)
        if B is None and "B" in want:
            B = mk(3 * self.N)
        if p is None and "p" in want:
            p = mk(self.N)
        if rho is None and "rho" in want:
            rho = mk(self.N)
        mhs_fields(self.h, B, p, rho, self.dtype, self.N, host=host, wait=wait)
        if host and not wait:
            # the copies are still in flight: the pinned buffers must outlive them even if the caller drops the result
            self._inflight = getattr(self, "_inflight", []) + [B, p, rho]
        shp = (self.nz, self.ny, self.nx)
        return (None if B is None else B.view(3, *shp), None if p is None else p.view(shp),
                None if rho is None else rho.view(shp))

    def diagnostics(self, B, want=("absB", "J", "absJ")):
        """|B|, j = curl B / mu0, |j| of the field mhs_fields returned (B: 3N device tensor or its (3, nz, ny, nx) view)."""
        mk = lambda n: torch.empty(n, dtype=self.dtype, device="cuda")
        aB = mk(self.N) if "absB" in want else None
        J = mk(3 * self.N) if "J" in want else None
        aJ = mk(self.N) if "absJ" in want else None
        _check(self.h, lib().mhs_diagnostics(self.h, _dptr(B.reshape(-1), self.dtype, 3 * self.N), _dptr(aB, self.dtype, self.N),
                                             _dptr(J, self.dtype, 3 * self.N), _dptr(aJ, self.dtype, self.N)))
        shp = (self.nz, self.ny, self.nx)
        return (None if aB is None else aB.view(shp), None if J is None else J.view(3, *shp), None if aJ is None else aJ.view(shp))

    def fieldlines(self, B, seeds, step, max_points, direction=1, bmin=0.0):
        """Field lines through `seeds` ((n, 3) device tensor of x, y, z) of the field mhs_fields returned.
        -> (lines (n, max_points, 3), npoints (n,) int32), device tensors; points beyond npoints[s] are NaN."""
        n = int(seeds.shape[0])
        lines = torch.full((n, max_points, 3), float("nan"), dtype=self.dtype, device="cuda")
        npts = torch.zeros(n, dtype=torch.int32, device="cuda")
        _check(self.h, lib().mhs_fieldlines(self.h, _dptr(B.reshape(-1), self.dtype, 3 * self.N), n,
                                            _dptr(seeds.reshape(-1), self.dtype, 3 * n), float(step), int(max_points),
                                            int(direction), float(bmin), C.c_void_p(lines.data_ptr()), C.c_void_p(npts.data_ptr())))
        return lines, npts

    def get_potential(self, out=None):
        if out is None:
            out = torch.empty((self.nz, self.ny, self.nx), dtype=self.dtype, device="cuda")
        mhs_get_potential(self.h, out, self.dtype, self.N)
        return out

    def get_boundary(self, out=None, host=False):
        """P(x, y, 0) of the last boundary solve, (ny, nx); host=True: into a pinned host tensor."""
        if out is None:
            out = torch.empty((self.ny, self.nx), dtype=self.dtype, device="cpu" if host else "cuda", pin_memory=host)
        fn = lib().mhs_get_boundary_host if not out.is_cuda else lib().mhs_get_boundary
        _check(self.h, fn(self.h, _dptr(out, self.dtype, self.nx * self.ny, "cuda" if out.is_cuda else "cpu")))
        return out

    def set_potential(self, P):
        mhs_set_potential(self.h, P, self.dtype, self.N)

    def set_wall_data(self, G):
        """Dirichlet data on the faces declared MHS_BC_DIRICHLET_DATA (Solver(..., bc=(sides, top))): G dense (nz, ny, nx) device tensor."""
        mhs_set_wall_data(self.h, G.reshape(-1), self.dtype, self.N)

    def profile(self):
        return mhs_get_profile(self.h)

    def reset_profile(self):
        mhs_reset_profile(self.h)

    def set_profiling(self, level):
        _check(self.h, lib().mhs_set_profiling(self.h, int(level)))

    # -- operator-level access (tests / micro-benchmarks)
    def num_levels(self, dim=3):
        return lib().mhs_num_levels(self.h, dim)

    def level_dims(self, dim, level):
        a, b, c = C.c_int(), C.c_int(), C.c_int()
        _check(self.h, lib().mhs_level_dims(self.h, dim, level, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def _shape(self, dim, level):
        nx, ny, nz = self.level_dims(dim, level)
        return (nz, ny, nx) if dim == 3 else (ny, nx)

    def level_set(self, dim, level, which, t):
        shp = self._shape(dim, level)
        _check(self.h, lib().mhs_level_set(self.h, dim, level, which, _dptr(t, self.dtype, int(np.prod(shp)))))

    def level_get(self, dim, level, which):
        shp = self._shape(dim, level)
        out = torch.empty(shp, dtype=self.dtype, device="cuda")
        _check(self.h, lib().mhs_level_get(self.h, dim, level, which, C.c_void_p(out.data_ptr())))
        return out

    def op_smooth(self, dim, level, sweeps=1):
        _check(self.h, lib().mhs_op_smooth(self.h, dim, level, sweeps))

    def op_residual(self, dim, level):
        _check(self.h, lib().mhs_op_residual(self.h, dim, level))

    def op_restrict(self, dim, level):
        _check(self.h, lib().mhs_op_restrict(self.h, dim, level))

    def op_prolong(self, dim, level):
        _check(self.h, lib().mhs_op_prolong(self.h, dim, level))

    def op_vcycle(self, dim, level):
        _check(self.h, lib().mhs_op_vcycle(self.h, dim, level))

    def op_resnorm(self, dim, level):
        v = C.c_double()
        _check(self.h, lib().mhs_op_resnorm(self.h, dim, level, C.byref(v)))
        return v.value
