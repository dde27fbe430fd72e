"""Seeded synthetic workloads (BASELINE.json configs 0-4 + the 2D-only 4097^2 case).

This module serves BOTH the oracle-side tests and the CUDA path and therefore holds none of
the method's arithmetic: it only produces inputs -- grids, the profile f(z) sampled at the
nodes, the magnetogram Bz0(x,y) and the background atmosphere.  numpy only; it imports neither
`oracle` nor the CUDA binding.

The paper uses no dataset: its examples are sums of analytic Gaussian flux sources on a
Dirichlet box.  BASELINE.json's configs keep that structure; the recipe
(readings C16-C19) is

  * generator: splitmix64, counter based, seed = 13076720 + config index;
    uniform(a,b) = a + (b-a) * (top 53 bits) / 2^53;
  * per patch, in order: amplitude A ~ U(-1,1), sigma ~ U(lo,hi), x0 ~ U(.15,.85) Lx,
    y0 ~ U(.15,.85) Ly (sources stay off the walls);
  * Bz0 = sum_k A_k exp(-r_k^2 / (2 sigma_k^2))  (BASELINE "sigma"; C17);
  * config 3 adds 1e-3 * U(-1,1) white noise per node, drawn after the patches in index order;
  * "net flux zeroed": subtract the arithmetic mean over all nx*ny nodes (C18);
  * f(z) = a exp(-kappa z) at the nodes z_k = k Lz/(nz-1);  xi(z) = -f(z)  (C1);
  * mu0 = 1/2, g = 1, p_b = rho_b = exp(-z)  (the paper's T_b = 1 layer; C16).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_MASK = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15
SEED_BASE = 13076720


def _mix64(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


class SplitMix64:
    """Counter-based splitmix64: draw n is mix(seed + (n+1)*gamma)."""

    def __init__(self, seed: int):
        self.seed = seed & _MASK
        self.count = 0

    def uniform(self, lo: float, hi: float, n: int | None = None):
        m = 1 if n is None else int(n)
        with np.errstate(over="ignore"):
            ctr = np.arange(self.count + 1, self.count + m + 1, dtype=np.uint64)
            z = _mix64(np.uint64(self.seed) + ctr * np.uint64(_GAMMA))
        self.count += m
        u = (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        v = lo + (hi - lo) * u
        return float(v[0]) if n is None else v


@dataclass
class Workload:
    """One synthetic problem: everything mhs_create / mhs_solve_* / mhs_fields need."""
    name: str
    nx: int
    ny: int
    nz: int
    Lx: float
    Ly: float
    Lz: float
    alpha: float
    a: float
    kappa: float
    dtype: str = "f64"
    n_pre: int = 2
    n_post: int = 2
    omega: float = 2.0 / 3.0
    tol: float = 1e-10
    max_cycles: int = 100
    mu0: float = 0.5
    g: float = 1.0
    Bz0: np.ndarray = field(default=None, repr=False)     # (ny, nx) float64
    f: np.ndarray = field(default=None, repr=False)       # (nz,)
    p_b: np.ndarray = field(default=None, repr=False)     # (nz,)
    rho_b: np.ndarray = field(default=None, repr=False)   # (nz,)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def L(self):
        return (self.Lx, self.Ly, self.Lz)

    @property
    def npoints(self):
        return self.nx * self.ny * self.nz


def gaussian_patches(nx, ny, Lx, Ly, amps, sigmas, x0s, y0s) -> np.ndarray:
    x = np.linspace(0.0, Lx, nx)[None, :]
    y = np.linspace(0.0, Ly, ny)[:, None]
    out = np.zeros((ny, nx))
    for A, s, x0, y0 in zip(amps, sigmas, x0s, y0s):
        out += A * np.exp(-((x - x0) ** 2 + (y - y0) ** 2) / (2.0 * s * s))
    return out


def random_patches(rng: SplitMix64, n, nx, ny, Lx, Ly, sig_lo, sig_hi) -> np.ndarray:
    amps, sigmas, x0s, y0s = [], [], [], []
    for _ in range(n):
        amps.append(rng.uniform(-1.0, 1.0))
        sigmas.append(rng.uniform(sig_lo, sig_hi))
        x0s.append(rng.uniform(0.15, 0.85) * Lx)
        y0s.append(rng.uniform(0.15, 0.85) * Ly)
    return gaussian_patches(nx, ny, Lx, Ly, amps, sigmas, x0s, y0s)


def profile(nz, Lz, a, kappa) -> np.ndarray:
    z = np.linspace(0.0, Lz, nz)
    return a * np.exp(-kappa * z) if a != 0.0 else np.zeros(nz)


def atmosphere(nz, Lz):
    z = np.linspace(0.0, Lz, nz)
    return np.exp(-z), np.exp(-z)


def _finish(w: Workload) -> Workload:
    w.f = profile(w.nz, w.Lz, w.a, w.kappa)
    w.p_b, w.rho_b = atmosphere(w.nz, w.Lz)
    return w


# name -> (grid, domain, alpha, a, kappa, n_patches, sigma range, extras)
_SPECS = {
    0: dict(n=(33, 33, 33), L=(1.0, 1.0, 1.0), alpha=0.5, a=0.0, kappa=0.0),
    1: dict(n=(129, 129, 129), L=(1.0, 1.0, 1.0), alpha=0.5, a=0.5, kappa=5.0, patches=4, sig=(0.03, 0.08)),
    2: dict(n=(257, 257, 257), L=(1.0, 1.0, 1.0), alpha=1.0, a=1.0, kappa=10.0, patches=16, sig=(0.02, 0.06)),
    3: dict(n=(513, 513, 513), L=(1.0, 1.0, 1.0), alpha=0.8, a=0.8, kappa=8.0, patches=64, sig=(0.02, 0.06),
            noise=1e-3, n_pre=3, n_post=3, tol=1e-9),
    4: dict(n=(1025, 1025, 257), L=(4.0, 4.0, 1.0), alpha=1.5, a=2.0, kappa=20.0, patches=256, sig=(0.01, 0.05),
            dtype="f32", tol=1e-6),
}


def config(index: int, shrink: int = 1, replica: int = 0) -> Workload:
    """BASELINE.json `configs[index]`.  `shrink` = 2^s divides the number of intervals per axis
    (same domain, same sources) -- used by parity tests that need an oracle-sized version of
    the big configs; shrink=1 is the configuration itself.  `replica` r > 0 draws an independent
    magnetogram of the same recipe (seed + 1000003 r): one per rank in multi-GPU replica runs."""
    s = _SPECS[index]
    nx, ny, nz = [(m - 1) // shrink + 1 for m in s["n"]]
    Lx, Ly, Lz = s["L"]
    w = Workload(name="config%d" % index + ("" if shrink == 1 else "/%d" % shrink), nx=nx, ny=ny,
                 nz=nz, Lx=Lx, Ly=Ly, Lz=Lz, alpha=s["alpha"], a=s["a"], kappa=s["kappa"],
                 dtype=s.get("dtype", "f64"), n_pre=s.get("n_pre", 2), n_post=s.get("n_post", 2),
                 tol=s.get("tol", 1e-10))
    if index == 0:
        # one bipole, deterministic (BASELINE configs[0]); no flux zeroing needed (C18/C19)
        w.Bz0 = gaussian_patches(nx, ny, Lx, Ly, [1.0, -1.0], [0.1, 0.1], [0.4, 0.6], [0.5, 0.5])
    else:
        rng = SplitMix64(SEED_BASE + index + 1000003 * replica)
        bz = random_patches(rng, s["patches"], nx, ny, Lx, Ly, *s["sig"])
        if "noise" in s:
            bz = bz + s["noise"] * rng.uniform(-1.0, 1.0, nx * ny).reshape(ny, nx)
        w.Bz0 = bz - bz.mean()
    return _finish(w)


def boundary_only(n: int = 4097, L: float = 4.0, patches: int = 256, dtype: str = "f32") -> Workload:
    """The 2D-only timing case of configs[4]: eq (11) on an n x n plane (domain [0,L]^2, same
    patch recipe, seed index 5).  nz = 1: a boundary-only context (include/mhs.h, mhs_create)."""
    rng = SplitMix64(SEED_BASE + 5)
    bz = random_patches(rng, patches, n, n, L, L, 0.01, 0.05)
    w = Workload(name="boundary%d" % n, nx=n, ny=n, nz=1, Lx=L, Ly=L, Lz=1.0, alpha=0.0, a=0.0,
                 kappa=0.0, dtype=dtype, tol=1e-6 if dtype == "f32" else 1e-10)
    w.Bz0 = bz - bz.mean()
    return _finish(w)


def small(nx=17, ny=33, nz=9, L=(1.0, 2.0, 0.5), alpha=0.7, a=0.6, kappa=4.0, patches=3,
          seed=99, n_pre=2, n_post=2) -> Workload:
    """A ragged, anisotropic little problem (different extents and spacings per axis) for tests."""
    rng = SplitMix64(SEED_BASE + seed)
    w = Workload(name="small%dx%dx%d" % (nx, ny, nz), nx=nx, ny=ny, nz=nz, Lx=L[0], Ly=L[1], Lz=L[2],
                 alpha=alpha, a=a, kappa=kappa, n_pre=n_pre, n_post=n_post)
    bz = random_patches(rng, patches, nx, ny, L[0], L[1], 0.08, 0.2)
    w.Bz0 = bz - bz.mean()
    return _finish(w)


def random_field(shape, seed: int, zero_boundary: bool = True) -> np.ndarray:
    """Seeded U(-1,1) array (test vectors for operator-level parity)."""
    rng = SplitMix64(SEED_BASE + 1000 + seed)
    a = rng.uniform(-1.0, 1.0, int(np.prod(shape))).reshape(shape)
    if zero_boundary:
        for ax in range(a.ndim):
            sl = [slice(None)] * a.ndim
            sl[ax] = 0
            a[tuple(sl)] = 0.0
            sl[ax] = -1
            a[tuple(sl)] = 0.0
    return a


def wall_data(w: "Workload", amp: float = 0.3, seed: int = 0) -> np.ndarray:
    """Dirichlet data for P on the side and top faces ("other elliptic equations can be defined on the other
    boundaries" -- their solutions would be such data): a smooth seeded function sampled on the whole (nz, ny, nx) grid; only its
    values on the side and top boundary nodes are used by the solver.  No method arithmetic here: just the samples."""
    rng = SplitMix64(SEED_BASE + 5000 + seed)
    k1, k2, k3, ph1, ph2 = (float(v) for v in rng.uniform(0.5, 2.5, 5))
    z = np.linspace(0.0, w.Lz, w.nz)[:, None, None]
    y = np.linspace(0.0, w.Ly, w.ny)[None, :, None]
    x = np.linspace(0.0, w.Lx, w.nx)[None, None, :]
    return amp * (np.sin(k1 * x / w.Lx * np.pi + ph1) * np.cos(k2 * y / w.Ly * np.pi + ph2) * np.exp(-k3 * z / w.Lz) + 0.25)


# ------------------------------------------------------------------------------------------------
# The paper's own examples (section 3): a second, fully analytic test-bed.
# ------------------------------------------------------------------------------------------------
def paper_atmosphere(z: np.ndarray, T_cor: float = 150.0, g: float = 1.0):
    """Background atmosphere of PAPER.md:123-132: T_b = 1 (z <= 5), T_cor^((z-5)/5) (5 < z <= 10), T_cor (z > 10);
    p_b solves dp_b/dz = -p_b g / T_b with p_b(0) = 1 (closed form per layer), rho_b = p_b / T_b."""
    z = np.asarray(z, dtype=np.float64)
    a = np.log(T_cor) / 5.0
    T = np.where(z <= 5.0, 1.0, np.where(z <= 10.0, np.exp(a * (np.clip(z, 5.0, 10.0) - 5.0)), T_cor))
    # integral of dz / T_b from 0 to z
    I1 = np.minimum(z, 5.0)
    I2 = (1.0 - np.exp(-a * (np.clip(z, 5.0, 10.0) - 5.0))) / a
    I3 = np.maximum(z - 10.0, 0.0) / T_cor
    p = np.exp(-g * (I1 + I2 + I3))
    return p, p / T


def paper_example(case: str = "force_free", n: int = 129, alpha: float | None = None) -> Workload:
    """PAPER.md:134-156.  Domain [-5.5, 5.5]^2 x [0, 12] (hx = hy != hz), three Gaussian sources B_z = B0 exp(-r^2/l^2),
    l = 0.3: +1 at (1.5, 1.5), -0.5 at (-1.5, -1.5) and (1.5, -1.5); alpha = 0.4.
      "force_free": xi = 0 (section 3.1);  "xi1": xi = 0.7 exp(-0.2 z) (eq 12);  "xi2": xi = [0.7 + 0.3 sin(pi z)] exp(-0.1 z)
      (eq 13).  f = -xi (C1).  Section 3.2 does not restate its sources or its alpha: the sources of 3.1 are assumed, and
      alpha defaults to 0.4 for the force-free case (the paper's) and to 0.2 for xi1, xi2 (ours).  The reason: with alpha = 0.4
      eq (8) is close to indefinite already for xi = 0 (alpha^2 = 0.16 against a smallest Laplacian eigenvalue of 0.232), and
      with 1 - xi down to 0.3 (xi1) or 0.05 (xi2) near the base it IS indefinite: V-cycles diverge, for the oracle and the
      library alike (the library reports MHS_ERR_INDEFINITE)."""
    if alpha is None:
        alpha = 0.4 if case == "force_free" else 0.2
    w = Workload(name="paper_%s_%d" % (case, n), nx=n, ny=n, nz=n, Lx=11.0, Ly=11.0, Lz=12.0, alpha=alpha, a=0.0, kappa=0.0)
    x = np.linspace(-5.5, 5.5, n)[None, :]
    y = np.linspace(-5.5, 5.5, n)[:, None]
    bz = np.zeros((n, n))
    for A, x0, y0 in ((1.0, 1.5, 1.5), (-0.5, -1.5, -1.5), (-0.5, 1.5, -1.5)):
        bz += A * np.exp(-((x - x0) ** 2 + (y - y0) ** 2) / 0.3 ** 2)
    w.Bz0 = bz
    z = np.linspace(0.0, 12.0, n)
    if case == "force_free":
        xi = np.zeros(n)
    elif case == "xi1":
        xi = 0.7 * np.exp(-0.2 * z)
    elif case == "xi2":
        xi = (0.7 + 0.3 * np.sin(np.pi * z)) * np.exp(-0.1 * z)
    else:
        raise ValueError(case)
    w.f = -xi
    w.p_b, w.rho_b = paper_atmosphere(z)
    return w
