"""ctypes front end of the CPU oracle (oracle/mhs_oracle.c) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; the product (paper_1307_6720_b200) never does, and this package never
imports the product.  Arrays are numpy float64, C-ordered with shape (nz, ny, nx) [3D] or
(ny, nx) [2D], i.e. x fastest in memory as in PAPER.md:214-216.

Every wrapper is argument marshalling only; the arithmetic lives in mhs_oracle.c, each function
there citing the passage of PAPER.md (or the DESIGN.md reading) it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhs_oracle.c")
_LIB = os.path.join(_HERE, "libmhs_oracle.so")
_lock = threading.Lock()
_lib = None

_d = C.c_double
_i = C.c_int
_p = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    """Compile mhs_oracle.c with gcc (-O2, OpenMP) into oracle/libmhs_oracle.so."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + ".%d.tmp" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
        os.replace(tmp, _LIB)
        return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_num_threads.restype = _i
        L.orc_is_coarsest.restype = _i
        L.orc_is_coarsest.argtypes = [_i] * 5
        L.orc_dense_solve.restype = _i
        L.orc_dense_solve.argtypes = [_i, _p, _p]
        g3 = [_i, _i, _i, _d, _d, _d]
        L.orc_apply3.argtypes = g3 + [_p, _d, _p, _p]
        L.orc_residual3.argtypes = g3 + [_p, _d, _p, _p, _p]
        L.orc_jacobi3.argtypes = g3 + [_p, _d, _d, _p, _p, _p]
        L.orc_restrict3.argtypes = [_i, _i, _i, _p, _p]
        L.orc_prolong_add3.argtypes = [_i, _i, _i, _p, _p]
        L.orc_norm3.restype = _d
        L.orc_norm3.argtypes = [_i, _i, _i, _p]
        L.orc_resnorm3.restype = _d
        L.orc_resnorm3.argtypes = g3 + [_p, _d, _p, _p]
        L.orc_direct3.restype = _i
        L.orc_direct3.argtypes = g3 + [_p, _d, _p, _p]
        L.orc_vcycle3.restype = _i
        L.orc_vcycle3.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _i, _p, _p]
        L.orc_solve3.restype = _i
        L.orc_solve3.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _d, _i, _p, _p, _p, _p, _i]
        L.orc_solve_interior.restype = _i
        L.orc_solve_interior.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _d, _i, _p, _p, _p, _i]
        g2 = [_i, _i, _d, _d]
        L.orc_apply2.argtypes = g2 + [_p, _p]
        L.orc_residual2.argtypes = g2 + [_p, _p, _p]
        L.orc_jacobi2.argtypes = g2 + [_d, _p, _p, _p]
        L.orc_restrict2.argtypes = [_i, _i, _p, _p]
        L.orc_prolong_add2.argtypes = [_i, _i, _p, _p]
        L.orc_norm2.restype = _d
        L.orc_norm2.argtypes = [_i, _i, _p]
        L.orc_resnorm2.restype = _d
        L.orc_resnorm2.argtypes = g2 + [_p, _p]
        L.orc_direct2.restype = _i
        L.orc_direct2.argtypes = g2 + [_p, _p]
        L.orc_vcycle2.restype = _i
        L.orc_vcycle2.argtypes = g2 + [_d, _i, _i, _i, _i, _p, _p]
        L.orc_solve2.restype = _i
        L.orc_solve2.argtypes = g2 + [_d, _i, _i, _i, _d, _i, _p, _p, _p, _p, _i]
        L.orc_solve_boundary.restype = _i
        L.orc_solve_boundary.argtypes = g2 + [_p, _d, _i, _i, _i, _d, _i, _p, _p, _p, _i]
        L.orc_fields.argtypes = g3 + [_d, _p, _p, _p, _p, _d, _d, _p, _p, _p, _p, _p, _p]
        L.orc_diagnostics.argtypes = g3 + [_d, _p, _p, _p, _p, _p, _p, _p, _p]
        L.orc_diagnostics.restype = None
        L.orc_zline3.argtypes = g3 + [_p, _d, _d, _p, _p, _p]
        L.orc_zline3.restype = None
        L.orc_vcycle3s.restype = _i
        L.orc_vcycle3s.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _i, _i, _p, _p]
        L.orc_fmg_interior.restype = _i
        L.orc_fmg_interior.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _i, _i, _p]
        L.orc_solve_interior_opt.restype = _i
        L.orc_solve_interior_opt.argtypes = g3 + [_p, _d, _d, _i, _i, _i, _i, _i, _d, _i, _p, _p, _p, _i]
        L.orc_fieldlines.argtypes = g3 + [_p, _p, _p, _i, _p, _d, _i, _i, _d, _p, C.POINTER(C.c_int)]
        L.orc_fieldlines.restype = None
        _lib = L
    return _lib


def _a(x):
    """float64 C-contiguous view/copy."""
    return np.ascontiguousarray(x, dtype=np.float64)


def _ptr(x):
    return None if x is None else x.ctypes.data_as(_p)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def is_coarsest(nx, ny, nz, level, max_levels=0) -> bool:
    return bool(lib().orc_is_coarsest(nx, ny, nz, level, max_levels))


def dense_solve(A, b):
    A = _a(A).copy(); b = _a(b).copy()
    rc = lib().orc_dense_solve(b.size, _ptr(A), _ptr(b))
    if rc:
        raise ArithmeticError("zero pivot")
    return b


# ------------------------------------------------------------------ 3D -----------------
def _g3(u, Lxyz):
    nz, ny, nx = u.shape
    Lx, Ly, Lz = Lxyz
    return nx, ny, nz, Lx / (nx - 1), Ly / (ny - 1), Lz / (nz - 1)


def apply3(u, c, alpha, Lxyz):
    u = _a(u); c = _a(c); out = np.empty_like(u)
    lib().orc_apply3(*_g3(u, Lxyz), _ptr(c), alpha, _ptr(u), _ptr(out))
    return out


def residual3(u, rhs, c, alpha, Lxyz):
    u = _a(u); c = _a(c); rhs = None if rhs is None else _a(rhs); r = np.empty_like(u)
    lib().orc_residual3(*_g3(u, Lxyz), _ptr(c), alpha, _ptr(u), _ptr(rhs), _ptr(r))
    return r


def jacobi3(u, rhs, c, alpha, omega, Lxyz):
    u = _a(u); c = _a(c); rhs = None if rhs is None else _a(rhs); un = np.empty_like(u)
    lib().orc_jacobi3(*_g3(u, Lxyz), _ptr(c), alpha, omega, _ptr(u), _ptr(rhs), _ptr(un))
    return un


def restrict3(r):
    r = _a(r); nz, ny, nx = r.shape
    rc = np.empty(((nz - 1) // 2 + 1, (ny - 1) // 2 + 1, (nx - 1) // 2 + 1))
    lib().orc_restrict3(nx, ny, nz, _ptr(r), _ptr(rc))
    return rc


def prolong_add3(ec, u):
    ec = _a(ec); u = _a(u).copy(); nz, ny, nx = u.shape
    lib().orc_prolong_add3(nx, ny, nz, _ptr(ec), _ptr(u))
    return u


def norm3(r):
    r = _a(r); nz, ny, nx = r.shape
    return float(lib().orc_norm3(nx, ny, nz, _ptr(r)))


def resnorm3(u, rhs, c, alpha, Lxyz):
    u = _a(u); c = _a(c); rhs = None if rhs is None else _a(rhs)
    return float(lib().orc_resnorm3(*_g3(u, Lxyz), _ptr(c), alpha, _ptr(u), _ptr(rhs)))


def direct3(u, rhs, c, alpha, Lxyz):
    u = _a(u).copy(); c = _a(c); rhs = None if rhs is None else _a(rhs)
    if lib().orc_direct3(*_g3(u, Lxyz), _ptr(c), alpha, _ptr(u), _ptr(rhs)):
        raise ArithmeticError("coarse solve failed")
    return u


def vcycle3(u, rhs, c, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, level=0):
    u = _a(u).copy(); c = _a(c); rhs = None if rhs is None else _a(rhs)
    if lib().orc_vcycle3(*_g3(u, Lxyz), _ptr(c), alpha, omega, n_pre, n_post, level, max_levels,
                         _ptr(u), _ptr(rhs)):
        raise ArithmeticError("coarse solve failed")
    return u


def solve3(u, rhs, c, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0,
           tol=1e-10, max_cycles=100, r0=0.0):
    u = _a(u).copy(); c = _a(c); rhs = None if rhs is None else _a(rhs)
    nz, ny, nx = u.shape
    hist = np.zeros(max(max_cycles, 1)); r0c = C.c_double(r0)
    n = lib().orc_solve3(nx, ny, nz, *Lxyz, _ptr(c), alpha, omega, n_pre, n_post, max_levels, tol,
                         max_cycles, _ptr(u), _ptr(rhs), C.cast(C.byref(r0c), _p), _ptr(hist),
                         hist.size)
    if n < 0:
        raise ArithmeticError("coarse solve failed")
    return u, dict(cycles=n, r0=r0c.value, history=hist[:n].copy())


def solve_interior(P, f, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0,
                   tol=1e-10, max_cycles=100, r0=0.0):
    """PAPER.md:100 (step 3).  P carries the bottom-plane data; returns (P, info)."""
    P = _a(P).copy(); f = _a(f)
    nz, ny, nx = P.shape
    hist = np.zeros(max(max_cycles, 1)); r0c = C.c_double(r0)
    n = lib().orc_solve_interior(nx, ny, nz, *Lxyz, _ptr(f), alpha, omega, n_pre, n_post,
                                 max_levels, tol, max_cycles, _ptr(P),
                                 C.cast(C.byref(r0c), _p), _ptr(hist), hist.size)
    if n < 0:
        raise ArithmeticError("coarse solve failed")
    return P, dict(cycles=n, r0=r0c.value, history=hist[:n].copy())


# ------------------------------------------------------------------ 2D -----------------
def _g2(u, Lxy):
    ny, nx = u.shape
    return nx, ny, Lxy[0] / (nx - 1), Lxy[1] / (ny - 1)


def apply2(u, Lxy):
    u = _a(u); out = np.empty_like(u)
    lib().orc_apply2(*_g2(u, Lxy), _ptr(u), _ptr(out))
    return out


def residual2(u, rhs, Lxy):
    u = _a(u); rhs = None if rhs is None else _a(rhs); r = np.empty_like(u)
    lib().orc_residual2(*_g2(u, Lxy), _ptr(u), _ptr(rhs), _ptr(r))
    return r


def jacobi2(u, rhs, omega, Lxy):
    u = _a(u); rhs = None if rhs is None else _a(rhs); un = np.empty_like(u)
    lib().orc_jacobi2(*_g2(u, Lxy), omega, _ptr(u), _ptr(rhs), _ptr(un))
    return un


def restrict2(r):
    r = _a(r); ny, nx = r.shape
    rc = np.empty(((ny - 1) // 2 + 1, (nx - 1) // 2 + 1))
    lib().orc_restrict2(nx, ny, _ptr(r), _ptr(rc))
    return rc


def prolong_add2(ec, u):
    ec = _a(ec); u = _a(u).copy(); ny, nx = u.shape
    lib().orc_prolong_add2(nx, ny, _ptr(ec), _ptr(u))
    return u


def norm2(r):
    r = _a(r); ny, nx = r.shape
    return float(lib().orc_norm2(nx, ny, _ptr(r)))


def resnorm2(u, rhs, Lxy):
    u = _a(u); rhs = None if rhs is None else _a(rhs)
    return float(lib().orc_resnorm2(*_g2(u, Lxy), _ptr(u), _ptr(rhs)))


def direct2(u, rhs, Lxy):
    u = _a(u).copy(); rhs = None if rhs is None else _a(rhs)
    if lib().orc_direct2(*_g2(u, Lxy), _ptr(u), _ptr(rhs)):
        raise ArithmeticError("coarse solve failed")
    return u


def vcycle2(u, rhs, Lxy, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, level=0):
    u = _a(u).copy(); rhs = None if rhs is None else _a(rhs)
    if lib().orc_vcycle2(*_g2(u, Lxy), omega, n_pre, n_post, level, max_levels, _ptr(u), _ptr(rhs)):
        raise ArithmeticError("coarse solve failed")
    return u


def solve2(u, rhs, Lxy, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, tol=1e-10,
           max_cycles=100, r0=0.0):
    u = _a(u).copy(); rhs = None if rhs is None else _a(rhs)
    ny, nx = u.shape
    hist = np.zeros(max(max_cycles, 1)); r0c = C.c_double(r0)
    n = lib().orc_solve2(nx, ny, *Lxy, omega, n_pre, n_post, max_levels, tol, max_cycles, _ptr(u),
                         _ptr(rhs), C.cast(C.byref(r0c), _p), _ptr(hist), hist.size)
    if n < 0:
        raise ArithmeticError("coarse solve failed")
    return u, dict(cycles=n, r0=r0c.value, history=hist[:n].copy())


def solve_boundary(Bz0, Lxy, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, tol=1e-10,
                   max_cycles=100):
    """PAPER.md:98-99 (steps 1-2): returns (P(x,y,0), info)."""
    Bz0 = _a(Bz0); ny, nx = Bz0.shape
    u2 = np.empty_like(Bz0); hist = np.zeros(max(max_cycles, 1)); r0c = C.c_double(0.0)
    n = lib().orc_solve_boundary(nx, ny, *Lxy, _ptr(Bz0), omega, n_pre, n_post, max_levels, tol,
                                 max_cycles, _ptr(u2), C.cast(C.byref(r0c), _p), _ptr(hist),
                                 hist.size)
    if n < 0:
        raise ArithmeticError("coarse solve failed")
    return u2, dict(cycles=n, r0=r0c.value, history=hist[:n].copy())


# --------------------------------------------------------------- fields ----------------
def fields(P, f, alpha, Lxyz, p_b, rho_b, mu0=0.5, g=1.0, dfdz=None):
    """PAPER.md:102-113, eqs 9-10: returns (Bx, By, Bz, p, rho)."""
    P = _a(P); f = _a(f); p_b = _a(p_b); rho_b = _a(rho_b)
    dfdz = None if dfdz is None else _a(dfdz)
    nz, ny, nx = P.shape
    out = [np.empty_like(P) for _ in range(5)]
    lib().orc_fields(nx, ny, nz, *Lxyz, alpha, _ptr(f), _ptr(dfdz), _ptr(p_b), _ptr(rho_b), mu0, g,
                     _ptr(P), *[_ptr(o) for o in out])
    return tuple(out)


def diagnostics(Bx, By, Bz, Lxyz, mu0=0.5):
    """|B| and j = curl B / mu0 with |j| (eq 2; Figs 2, 4-7): returns (absB, jx, jy, jz, absJ)."""
    Bx = _a(Bx); By = _a(By); Bz = _a(Bz)
    nz, ny, nx = Bx.shape
    out = [np.empty_like(Bx) for _ in range(5)]
    lib().orc_diagnostics(nx, ny, nz, *Lxyz, mu0, _ptr(Bx), _ptr(By), _ptr(Bz), *[_ptr(o) for o in out])
    return tuple(out)


def fieldlines(Bx, By, Bz, Lxyz, seeds, step, max_points, direction=1, bmin=0.0):
    """RK4 field-line integration through the trilinearly interpolated nodal B (Figs 1, 4, 5).
    seeds: (n, 3) positions (x, y, z) in [0,Lx]x[0,Ly]x[0,Lz].  Returns (lines (n, max_points, 3), npoints (n,))."""
    Bx, By, Bz = _a(Bx), _a(By), _a(Bz)
    nz, ny, nx = Bx.shape
    seeds = _a(seeds).reshape(-1, 3)
    n = seeds.shape[0]
    lines = np.full((n, max_points, 3), np.nan)
    npts = np.zeros(n, dtype=np.int32)
    lib().orc_fieldlines(nx, ny, nz, *Lxyz, _ptr(Bx), _ptr(By), _ptr(Bz), n, _ptr(seeds), float(step), int(max_points),
                         int(direction), float(bmin), _ptr(lines), npts.ctypes.data_as(C.POINTER(C.c_int)))
    return lines, npts


# ---- solver variants: z-line Jacobi smoothing, full-multigrid start -------------------------------
def zline3(u, rhs, c, alpha, omega, Lxyz):
    """One weighted z-line Jacobi sweep: unew = u + omega T^-1 (rhs - L u), T = the z-tridiagonal part of L."""
    u = _a(u); c = _a(c); rhs = None if rhs is None else _a(rhs)
    un = np.empty_like(u)
    lib().orc_zline3(*_g3(u, Lxyz), _ptr(c), alpha, omega, _ptr(u), _ptr(rhs), _ptr(un))
    return un


def vcycle3s(u, rhs, c, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, level=0, smoother=0):
    u = _a(u).copy(); c = _a(c); rhs = None if rhs is None else _a(rhs)
    if lib().orc_vcycle3s(*_g3(u, Lxyz), _ptr(c), alpha, omega, n_pre, n_post, level, max_levels, smoother, _ptr(u), _ptr(rhs)):
        raise ArithmeticError("coarse solve failed")
    return u


def fmg_interior(P, f, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, smoother=0, n_fmg=1):
    """Full-multigrid initial guess for step 3 from the bottom-plane data in P (the interior of P is ignored)."""
    P = _a(P).copy(); f = _a(f)
    nz, ny, nx = P.shape
    if lib().orc_fmg_interior(nx, ny, nz, *Lxyz, _ptr(f), alpha, omega, n_pre, n_post, max_levels, smoother, n_fmg, _ptr(P)):
        raise ArithmeticError("coarse solve failed")
    return P


def solve_interior_opt(P, f, alpha, Lxyz, omega=2.0 / 3.0, n_pre=2, n_post=2, max_levels=0, smoother=0, fmg=0,
                       tol=1e-10, max_cycles=100, r0=0.0):
    P = _a(P).copy(); f = _a(f)
    nz, ny, nx = P.shape
    hist = np.zeros(max(max_cycles, 1)); r0c = C.c_double(r0)
    n = lib().orc_solve_interior_opt(nx, ny, nz, *Lxyz, _ptr(f), alpha, omega, n_pre, n_post, max_levels, smoother, fmg,
                                     tol, max_cycles, _ptr(P), C.cast(C.byref(r0c), _p), _ptr(hist), hist.size)
    if n < 0:
        raise ArithmeticError("coarse solve failed")
    return P, dict(cycles=n, r0=r0c.value, history=hist[:n].copy())
