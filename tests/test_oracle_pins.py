"""Pins for the CPU oracle (oracle/mhs_oracle.c): every function is checked against something
OTHER than itself -- closed forms of the discrete and continuous problems, Fourier symbols of the
multigrid components, invariants (symmetry, adjointness, div B = 0, force balance), a dense
Kronecker-product re-formulation on tiny grids (brute force) and numpy's LAPACK solve.

PAPER.md prints no numerical value of P, B, p or rho (figures only), so there is no golden
fixture from the paper; these pins (P1..P14 of SURVEY.md section 8(c) / DESIGN.md) replace it.
CPU only:  python -m pytest tests -m "not gpu".
"""
import numpy as np
import pytest

from paper_1307_6720_b200 import inputs

W23 = 2.0 / 3.0


# ----------------------------------------------------------------------- helpers -------------
def grid(n, L):
    return np.linspace(0.0, L, n)


def sinmode(n, m):
    """sin(m pi i/(n-1)), i = 0..n-1 (vanishes on both walls)."""
    return np.sin(m * np.pi * np.arange(n) / (n - 1))


def lam(n, L, m):
    """eigenvalue of -dxx on the mode m: (4/h^2) sin^2(k h/2), k = m pi/L."""
    h = L / (n - 1)
    return 4.0 / h**2 * np.sin(m * np.pi / L * h / 2.0) ** 2


def T1(n, h):
    """1-D second-difference matrix on the n-2 interior nodes."""
    m = n - 2
    return (np.diag(-2.0 * np.ones(m)) + np.diag(np.ones(m - 1), 1) + np.diag(np.ones(m - 1), -1)) / h**2


def R1(n):
    """1-D full weighting, fine n nodes -> coarse (n-1)/2+1 nodes, interior to interior."""
    nc = (n - 1) // 2 + 1
    R = np.zeros((nc - 2, n - 2))
    for I in range(1, nc - 1):
        for a, w in ((-1, 0.25), (0, 0.5), (1, 0.25)):
            R[I - 1, 2 * I + a - 1] = w
    return R


def kron3(Az, Ay, Ax):
    return np.kron(Az, np.kron(Ay, Ax))


def interior(a):
    return a[tuple(slice(1, -1) for _ in range(a.ndim))]


def embed(v, shape):
    out = np.zeros(shape)
    out[tuple(slice(1, -1) for _ in shape)] = v.reshape([s - 2 for s in shape])
    return out


# ----------------------------------------------------------------------- level rule ----------
def test_level_rule_counts(orc):
    def nlevels(nx, ny, nz, max_levels=0):
        l = 0
        while not orc.is_coarsest(nx, ny, nz, l, max_levels):
            nx, ny = (nx - 1) // 2 + 1, (ny - 1) // 2 + 1
            nz = (nz - 1) // 2 + 1 if nz > 1 else nz
            l += 1
        return l + 1, (nx, ny, nz)

    assert nlevels(33, 33, 33) == (5, (3, 3, 3))             # "33^3 ... 5 levels"
    assert nlevels(257, 257, 257) == (8, (3, 3, 3))
    assert nlevels(513, 513, 513) == (9, (3, 3, 3))
    assert nlevels(1025, 1025, 257) == (8, (9, 9, 3))        # config 4 coarsest 9x9x3
    assert nlevels(4097, 4097, 1) == (12, (3, 3, 1))         # 2D
    assert nlevels(17, 33, 9) == (3, (5, 9, 3))
    assert nlevels(25, 25, 13) == (3, (7, 7, 4))             # 12 -> 6 -> 3 intervals (odd: stop)
    assert nlevels(33, 33, 33, max_levels=2)[0] == 2


def test_dense_solve_vs_lapack(orc):
    rng = np.random.default_rng(7)
    for n in (1, 2, 7, 49):
        A = rng.standard_normal((n, n))
        if n > 1:
            A[0, 0] = 0.0  # forces a row exchange
        b = rng.standard_normal(n)
        np.testing.assert_allclose(orc.dense_solve(A, b), np.linalg.solve(A, b), rtol=1e-10, atol=1e-12)


# ----------------------------------------------------------------------- P4: smoother symbol -
@pytest.mark.parametrize("cconst", [1.0, 1.3])
def test_P4_jacobi_symbol_3d(orc, cconst):
    nx, ny, nz = 17, 33, 9
    L = (1.0, 2.0, 0.5)
    alpha, omega = 0.7, 0.8
    hx, hy, hz = [Lq / (n - 1) for Lq, n in zip(L, (nx, ny, nz))]
    c = np.full(nz, cconst)
    for (a, b, d) in [(1, 1, 1), (3, 5, 2), (15, 31, 7), (8, 1, 4)]:
        u = sinmode(nz, d)[:, None, None] * sinmode(ny, b)[None, :, None] * sinmode(nx, a)[None, None, :]
        lx, ly, lz = lam(nx, L[0], a), lam(ny, L[1], b), lam(nz, L[2], d)
        fac = 1.0 - omega * (cconst * (lx + ly) + lz - alpha**2) / (
            2 * cconst / hx**2 + 2 * cconst / hy**2 + 2 / hz**2 - alpha**2)
        un = orc.jacobi3(u, None, c, alpha, omega, L)
        np.testing.assert_allclose(un, fac * u, rtol=0, atol=2e-14)
        # operator symbol too: L u = (-c(lx+ly) - lz + alpha^2) u
        np.testing.assert_allclose(orc.apply3(u, c, alpha, L), (-cconst * (lx + ly) - lz + alpha**2) * u,
                                   rtol=0, atol=1e-9 * (lx + ly + lz))


def test_P4_jacobi_symbol_2d_and_rhs(orc):
    nx, ny = 33, 17
    L = (1.0, 3.0)
    hx, hy = L[0] / (nx - 1), L[1] / (ny - 1)
    u = sinmode(ny, 3)[:, None] * sinmode(nx, 5)[None, :]
    lx, ly = lam(nx, L[0], 5), lam(ny, L[1], 3)
    fac = 1.0 - W23 * (lx + ly) / (2 / hx**2 + 2 / hy**2)
    np.testing.assert_allclose(orc.jacobi2(u, None, W23, L), fac * u, atol=2e-14)
    # with rhs = L2 u the sweep must leave u unchanged (fixed point), boundary copied
    rhs = -(lx + ly) * u
    np.testing.assert_allclose(orc.jacobi2(u, rhs, W23, L), u, atol=1e-13)
    np.testing.assert_allclose(orc.residual2(u, rhs, L), 0 * u, atol=1e-9)
    # boundary branch: non-zero boundary values are passed through untouched
    v = inputs.random_field((ny, nx), 1, zero_boundary=False)
    vn = orc.jacobi2(v, None, W23, L)
    for sl in (np.s_[0, :], np.s_[-1, :], np.s_[:, 0], np.s_[:, -1]):
        assert np.array_equal(vn[sl], v[sl])


def test_jacobi3_boundary_branch_and_variable_c(orc):
    """PAPER.md:218 boundary branch; and the z-dependent coefficient sits on the right planes:
    for u = g(z) * sin*sin the sweep reduces to a 1-D formula in z with c_k on plane k."""
    nx, ny, nz = 9, 9, 17
    L = (1.0, 1.0, 2.0)
    hx, hy, hz = [Lq / (n - 1) for Lq, n in zip(L, (nx, ny, nz))]
    c = 1.0 + 0.8 * np.exp(-3.0 * grid(nz, L[2]))
    gz = np.cos(1.7 * grid(nz, L[2])) + 0.3
    sxy = sinmode(ny, 2)[:, None] * sinmode(nx, 3)[None, :]
    u = gz[:, None, None] * sxy[None]
    alpha, omega = 0.4, 0.6
    lxy = lam(nx, L[0], 3) + lam(ny, L[1], 2)
    un = orc.jacobi3(u, None, c, alpha, omega, L)
    exp = gz.copy()
    for k in range(1, nz - 1):
        Lu = -c[k] * lxy * gz[k] + (gz[k + 1] - 2 * gz[k] + gz[k - 1]) / hz**2 + alpha**2 * gz[k]
        D = -2 * c[k] / hx**2 - 2 * c[k] / hy**2 - 2 / hz**2 + alpha**2
        exp[k] = gz[k] - omega / D * Lu
    np.testing.assert_allclose(un, exp[:, None, None] * sxy[None], atol=1e-13)
    assert np.array_equal(un[0], u[0]) and np.array_equal(un[-1], u[-1])


# ----------------------------------------------------------------------- P5: transfer symbols
def test_P5_full_weighting_symbol(orc):
    nx, ny, nz = 17, 33, 9
    for (a, b, d) in [(1, 1, 1), (3, 7, 2), (7, 15, 3)]:
        r = sinmode(nz, d)[:, None, None] * sinmode(ny, b)[None, :, None] * sinmode(nx, a)[None, None, :]
        th = [np.pi * m / (n - 1) for m, n in ((a, nx), (b, ny), (d, nz))]
        fac = np.prod([np.cos(t / 2) ** 2 for t in th])
        cx, cy, cz = 9, 17, 5
        exp = fac * sinmode(cz, d)[:, None, None] * sinmode(cy, b)[None, :, None] * sinmode(cx, a)[None, None, :]
        np.testing.assert_allclose(orc.restrict3(r), exp, atol=1e-14)
    r2 = sinmode(ny, 5)[:, None] * sinmode(nx, 2)[None, :]
    fac = np.cos(np.pi * 5 / (ny - 1) / 2) ** 2 * np.cos(np.pi * 2 / (nx - 1) / 2) ** 2
    np.testing.assert_allclose(orc.restrict2(r2), fac * sinmode(17, 5)[:, None] * sinmode(9, 2)[None, :], atol=1e-14)
    # a constant interior residual restricts to the same constant away from the walls (weights sum to 1)
    ones = np.ones((9, 9, 9))
    assert np.allclose(orc.restrict3(ones)[1:-1, 1:-1, 1:-1], 1.0) and orc.restrict3(ones)[0].max() == 0.0


def test_P5_linear_interpolation_symbol(orc):
    nx, ny, nz = 17, 33, 9
    cx, cy, cz = 9, 17, 5
    a, b, d = 2, 5, 1
    ec = sinmode(cz, d)[:, None, None] * sinmode(cy, b)[None, :, None] * sinmode(cx, a)[None, None, :]

    def one_d(n, m):  # even nodes: the mode itself; odd nodes: cos(theta) * mode
        i = np.arange(n)
        th = np.pi * m / (n - 1)
        return np.where(i % 2 == 0, 1.0, np.cos(th)) * sinmode(n, m)

    exp = one_d(nz, d)[:, None, None] * one_d(ny, b)[None, :, None] * one_d(nx, a)[None, None, :]
    u0 = inputs.random_field((nz, ny, nx), 3, zero_boundary=False)
    got = orc.prolong_add3(ec, u0) - u0
    np.testing.assert_allclose(interior(got), interior(exp), atol=1e-14)
    # boundary nodes of u are not touched (correction acts on interior fine nodes only)
    bd = np.ones_like(got, bool); bd[1:-1, 1:-1, 1:-1] = False
    assert np.all(got[bd] == 0.0)
    e2 = sinmode(cy, b)[:, None] * sinmode(cx, a)[None, :]
    got2 = orc.prolong_add2(e2, np.zeros((ny, nx)))
    np.testing.assert_allclose(got2, one_d(ny, b)[:, None] * one_d(nx, a)[None, :], atol=1e-14)


# ----------------------------------------------------------------------- P6, P7 --------------
def test_P6_restriction_prolongation_adjoint(orc):
    nx, ny, nz = 17, 9, 33
    r = inputs.random_field((nz, ny, nx), 11)
    e = inputs.random_field((17, 5, 9), 12)
    lhs = 8.0 * np.sum(orc.restrict3(r) * e)
    rhs = np.sum(r * orc.prolong_add3(e, np.zeros_like(r)))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    r2 = inputs.random_field((ny, nx), 13)
    e2 = inputs.random_field((5, 9), 14)
    lhs = 4.0 * np.sum(orc.restrict2(r2) * e2)
    rhs = np.sum(r2 * orc.prolong_add2(e2, np.zeros_like(r2)))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_P7_operator_symmetric(orc):
    nx, ny, nz = 9, 17, 13
    L = (1.0, 0.7, 2.0)
    c = 1.0 + 0.9 * np.exp(-2.0 * grid(nz, L[2]))
    u = inputs.random_field((nz, ny, nx), 21)
    v = inputs.random_field((nz, ny, nx), 22)
    a = np.sum(orc.apply3(u, c, 0.9, L) * v)
    b = np.sum(u * orc.apply3(v, c, 0.9, L))
    assert abs(a - b) <= 1e-12 * abs(a)
    u2, v2 = u[3], v[3]
    a = np.sum(orc.apply2(u2, L[:2]) * v2); b = np.sum(u2 * orc.apply2(v2, L[:2]))
    assert abs(a - b) <= 1e-12 * abs(a)


# ----------------------------------------------------------------------- P8: brute force -----
def _dense_level(nx, ny, nz, hx, hy, hz, c, alpha):
    mx, my, mz = nx - 2, ny - 2, nz - 2
    Ix, Iy, Iz = np.eye(mx), np.eye(my), np.eye(mz)
    C = np.diag(c[1:-1])
    A = kron3(C, Iy, T1(nx, hx)) + kron3(C, T1(ny, hy), Ix) + kron3(T1(nz, hz), Iy, Ix) + alpha**2 * np.eye(mx * my * mz)
    return A


def _dense_vcycle(level, dims, h, c, alpha, omega, n1, n2, max_levels, v, rhs, orc):
    nx, ny, nz = dims
    A = _dense_level(nx, ny, nz, *h, c, alpha)
    if orc.is_coarsest(nx, ny, nz, level, max_levels):
        return np.linalg.solve(A, rhs)
    Dinv = 1.0 / np.diag(A)
    for _ in range(n1):
        v = v + omega * Dinv * (rhs - A @ v)
    r = rhs - A @ v
    R = kron3(R1(nz), R1(ny), R1(nx))
    cd = ((nx - 1) // 2 + 1, (ny - 1) // 2 + 1, (nz - 1) // 2 + 1)
    ec = _dense_vcycle(level + 1, cd, [2 * q for q in h], c[::2], alpha, omega, n1, n2, max_levels,
                       np.zeros(R.shape[0]), R @ r, orc)
    v = v + 8.0 * R.T @ ec
    for _ in range(n2):
        v = v + omega * Dinv * (rhs - A @ v)
    return v


@pytest.mark.parametrize("dims,L", [((9, 9, 9), (1.0, 1.0, 1.0)), ((9, 9, 5), (1.0, 1.3, 0.4)), ((5, 9, 3), (0.5, 1.0, 0.25))])
def test_P8_vcycle_equals_dense_matrix_formulation(orc, dims, L):
    nx, ny, nz = dims
    h = [Lq / (n - 1) for Lq, n in zip(L, dims)]
    f = 0.7 * np.exp(-2.5 * grid(nz, L[2]))
    c = 1.0 + f
    alpha = 0.8
    P = np.zeros((nz, ny, nx))
    P[0] = inputs.random_field((ny, nx), 31)                     # bottom Dirichlet data, zero edges
    rhs_eff = np.zeros((nz - 2, ny - 2, nx - 2))
    rhs_eff[0] = -P[0, 1:-1, 1:-1] / h[2] ** 2                    # boundary data moved to the rhs
    rhs_eff = rhs_eff.ravel()
    v = np.zeros_like(rhs_eff)
    A = _dense_level(nx, ny, nz, *h, c, alpha)
    exact = np.linalg.solve(A, rhs_eff)
    scale = np.abs(exact).max()
    for it in range(6):
        P = orc.vcycle3(P, None, c, alpha, L, omega=W23, n_pre=2, n_post=2)
        v = _dense_vcycle(0, dims, h, c, alpha, W23, 2, 2, 0, v, rhs_eff, orc)
        assert np.abs(interior(P).ravel() - v).max() <= 1e-14 * scale, it
        # residual norm agrees with the matrix residual
        assert abs(orc.resnorm3(P, None, c, alpha, L) - np.linalg.norm(rhs_eff - A @ v)) <= 1e-9 * np.linalg.norm(rhs_eff)
    # (i) MG limit == dense direct solve; and the oracle's own direct solve agrees with LAPACK
    Pc, info = orc.solve_interior(P, f, alpha, L, tol=1e-13, max_cycles=60)
    assert np.abs(interior(Pc).ravel() - exact).max() <= 1e-11 * scale
    P0 = np.zeros((nz, ny, nx)); P0[0] = Pc[0]
    np.testing.assert_allclose(interior(orc.direct3(P0, None, c, alpha, L)).ravel(), exact, atol=1e-13 * scale)


def test_P8_vcycle_2d_dense(orc):
    nx, ny = 9, 17
    L = (1.0, 1.5)
    hx, hy = L[0] / (nx - 1), L[1] / (ny - 1)

    def A2(nx, ny, hx, hy):
        return np.kron(np.eye(ny - 2), T1(nx, hx)) + np.kron(T1(ny, hy), np.eye(nx - 2))

    def V(level, nx, ny, hx, hy, v, rhs):
        A = A2(nx, ny, hx, hy)
        if orc.is_coarsest(nx, ny, 1, level, 0):
            return np.linalg.solve(A, rhs)
        Dinv = 1.0 / np.diag(A)
        for _ in range(2):
            v = v + W23 * Dinv * (rhs - A @ v)
        R = np.kron(R1(ny), R1(nx))
        ec = V(level + 1, (nx - 1) // 2 + 1, (ny - 1) // 2 + 1, 2 * hx, 2 * hy, np.zeros(R.shape[0]), R @ (rhs - A @ v))
        v = v + 4.0 * R.T @ ec
        for _ in range(2):
            v = v + W23 * Dinv * (rhs - A @ v)
        return v

    rhs = inputs.random_field((ny, nx), 41)
    u = np.zeros((ny, nx)); v = np.zeros((ny - 2) * (nx - 2))
    for it in range(5):
        u = orc.vcycle2(u, rhs, L)
        v = V(0, nx, ny, hx, hy, v, interior(rhs).ravel())
        assert np.abs(interior(u).ravel() - v).max() <= 1e-14 * np.abs(v).max()
    exact = np.linalg.solve(A2(nx, ny, hx, hy), interior(rhs).ravel())
    us, info = orc.solve2(np.zeros((ny, nx)), rhs, L, tol=1e-13, max_cycles=60)
    assert np.abs(interior(us).ravel() - exact).max() <= 1e-11 * np.abs(exact).max()
    np.testing.assert_allclose(interior(orc.direct2(np.zeros((ny, nx)), rhs, L)).ravel(), exact, atol=1e-13)


# ----------------------------------------------------------------------- P1, P2, P3 ----------
def _separable_Z(nz, hz, c, lxy, alpha):
    """Z_{k+1} - (2 + hz^2 (c_k lxy - alpha^2)) Z_k + Z_{k-1} = 0, Z_0 = 1, Z_{nz-1} = 0."""
    m = nz - 2
    M = np.zeros((m, m)); b = np.zeros(m)
    for k in range(1, nz - 1):
        M[k - 1, k - 1] = -(2.0 + hz**2 * (c[k] * lxy - alpha**2))
        if k > 1: M[k - 1, k - 2] = 1.0
        if k < nz - 2: M[k - 1, k] = 1.0
    b[0] = -1.0
    Z = np.zeros(nz); Z[0] = 1.0; Z[1:-1] = np.linalg.solve(M, b)
    return Z


def test_P1_discrete_closed_form_force_free(orc):
    nx, ny, nz = 33, 17, 33
    L = (1.0, 0.8, 1.2)
    alpha = 0.5
    hz = L[2] / (nz - 1)
    bottom = sinmode(ny, 1)[:, None] * sinmode(nx, 2)[None, :]
    lxy = lam(nx, L[0], 2) + lam(ny, L[1], 1)
    mu = np.arccosh(1.0 + hz**2 * (lxy - alpha**2) / 2.0)
    k = np.arange(nz)
    Z = np.sinh(mu * (nz - 1 - k)) / np.sinh(mu * (nz - 1))
    P = np.zeros((nz, ny, nx)); P[0] = bottom
    P, info = orc.solve_interior(P, np.zeros(nz), alpha, L, tol=1e-12, max_cycles=60)
    assert np.abs(P - Z[:, None, None] * bottom[None]).max() <= 5e-11
    assert info["history"][-1] <= 1e-12 * info["r0"]


def test_P2_discrete_separable_form_variable_coefficient(orc):
    nx, ny, nz = 17, 17, 33
    L = (1.0, 1.0, 1.0)
    alpha = 1.0
    f = 1.0 * np.exp(-10.0 * grid(nz, 1.0))                       # config-2 operator
    bottom = sinmode(ny, 2)[:, None] * sinmode(nx, 1)[None, :]
    lxy = lam(nx, 1.0, 1) + lam(ny, 1.0, 2)
    Z = _separable_Z(nz, 1.0 / (nz - 1), 1.0 + f, lxy, alpha)
    P = np.zeros((nz, ny, nx)); P[0] = bottom
    P, info = orc.solve_interior(P, f, alpha, L, tol=1e-12, max_cycles=80)
    assert np.abs(P - Z[:, None, None] * bottom[None]).max() <= 5e-11
    # a coefficient shifted by one plane (c_{k+1} used on plane k) must NOT pass
    Zbad = _separable_Z(nz, 1.0 / (nz - 1), np.roll(1.0 + f, -1), lxy, alpha)
    assert np.abs(P - Zbad[:, None, None] * bottom[None]).max() > 1e-3


def test_P3_boundary_poisson_closed_form(orc):
    nx, ny = 33, 65
    L = (1.0, 2.0)
    Bz0 = sinmode(ny, 3)[:, None] * sinmode(nx, 2)[None, :]
    P0, info = orc.solve_boundary(Bz0, L, tol=1e-12, max_cycles=60)
    lxy = lam(nx, L[0], 2) + lam(ny, L[1], 3)
    assert np.abs(P0 - Bz0 / lxy).max() <= 1e-12                   # sign of eq (11): P0 has Bz0's sign
    assert abs(info["r0"] - np.linalg.norm(interior(Bz0))) <= 1e-12 * info["r0"]


# ----------------------------------------------------------------------- P9: O(h^2) ----------
def test_P9_second_order_vs_continuous_solution(orc):
    L = (1.0, 1.0, 1.0)
    alpha = 0.5
    kx, ky = np.pi, 2 * np.pi
    l = np.sqrt(kx**2 + ky**2 - alpha**2)
    errs = []
    for n in (9, 17, 33, 65):
        x = grid(n, 1.0)
        bottom = np.sin(ky * x)[:, None] * np.sin(kx * x)[None, :]
        bottom[0] = bottom[-1] = 0.0; bottom[:, 0] = bottom[:, -1] = 0.0
        exact = (np.sinh(l * (1.0 - x)) / np.sinh(l))[:, None, None] * bottom[None]
        P = np.zeros((n, n, n)); P[0] = bottom
        P, _ = orc.solve_interior(P, np.zeros(n), alpha, L, tol=1e-11, max_cycles=60)
        errs.append(np.abs(P - exact).max())
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert 3.5 < ratios[-1] < 4.5 and ratios[-2] > 3.2, (errs, ratios)


def test_P9_manufactured_solution_with_rhs(orc):
    """u* = sin(pi x) sin(2 pi y) q(z), q = z(1-z)e^z, variable c(z): rhs = L_cont u*."""
    alpha = 0.9
    errs = []
    for n in (9, 17, 33, 65):
        x = grid(n, 1.0)
        z = x
        c = 1.0 + 0.5 * np.exp(-3.0 * z)
        q = z * (1 - z) * np.exp(z)
        qpp = np.exp(z) * (-z * z - 3 * z)                          # d2/dz2 [ (z - z^2) e^z ]
        sxy = np.sin(2 * np.pi * x)[:, None] * np.sin(np.pi * x)[None, :]
        ustar = q[:, None, None] * sxy[None]
        rhs = (c * (-(np.pi**2 + 4 * np.pi**2)) * q + qpp + alpha**2 * q)[:, None, None] * sxy[None]
        u, info = orc.solve3(np.zeros((n, n, n)), rhs, c, alpha, (1.0, 1.0, 1.0), tol=1e-11, max_cycles=80)
        errs.append(np.abs(u - ustar).max())
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert 3.6 < ratios[-1] < 4.4 and ratios[-2] > 3.3, (errs, ratios)


# ----------------------------------------------------------------------- fields pins ---------
def _analytic_P(n, L, alpha):
    """A smooth P (not a PDE solution) with analytic derivatives, zero on the side walls."""
    x, y, z = grid(n, L[0]), grid(n, L[1]), grid(n, L[2])
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
    a, b, d = np.pi / L[0], 2 * np.pi / L[1], 1.3
    sx, cx, sy, cy = np.sin(a * X), np.cos(a * X), np.sin(b * Y), np.cos(b * Y)
    ez = np.exp(-d * Z)
    P = sx * sy * ez
    Bx = alpha * (b * sx * cy * ez) + (-d * a * cx * sy * ez)
    By = -alpha * (a * cx * sy * ez) + (-d * b * sx * cy * ez)
    Bz = (a * a + b * b) * P
    dBz = ((a * a + b * b) * a * cx * sy * ez, (a * a + b * b) * b * sx * cy * ez, -d * Bz)
    return P, Bx, By, Bz, dBz


def test_fields_converge_to_analytic_formulas(orc):
    """B, p, rho from FD vs eqs 5, 9, 10 evaluated with analytic derivatives:
    error ~ h^2 at interior nodes AND on the bottom plane (one-sided z differences, C13)."""
    L = (1.0, 1.5, 0.8)
    alpha, mu0, g = 0.7, 0.5, 1.3
    errs = []
    for n in (17, 33, 65):
        z = grid(n, L[2])
        f = 0.6 * np.exp(-2.0 * z); dfdz = -1.2 * np.exp(-2.0 * z)
        p_b = np.exp(-z); rho_b = 2.0 * np.exp(-0.5 * z)
        P, Bx, By, Bz, dBz = _analytic_P(n, L, alpha)
        gBx, gBy, gBz, gp, grho = orc.fields(P, f, alpha, L, p_b, rho_b, mu0=mu0, g=g)
        xi, dxi = -f[:, None, None], -dfdz[:, None, None]
        p = p_b[:, None, None] - xi * Bz**2 / (2 * mu0)
        rho = rho_b[:, None, None] + (dxi * Bz**2 / (2 * mu0) + xi / mu0 * (Bx * dBz[0] + By * dBz[1] + Bz * dBz[2])) / g
        s = np.s_[0:-1, 1:-1, 1:-1]                                  # everything that is not side/top
        si = np.s_[0:-2, 2:-2, 2:-2]                                 # rho: grad Bz uses wall values B = 0 (C13), skip
        errs.append([np.abs(gBx[s] - Bx[s]).max(), np.abs(gBy[s] - By[s]).max(), np.abs(gBz[s] - Bz[s]).max(),
                     np.abs(gp[s] - p[s]).max(), np.abs(grho[si] - rho[si]).max()])
        # walls: B = 0, p = p_b, rho = rho_b (C13, C15)
        for arr in (gBx, gBy, gBz):
            assert arr[-1].max() == 0 and np.abs(arr[:, 0]).max() == 0 and np.abs(arr[:, :, -1]).max() == 0
        assert np.array_equal(gp[-1], np.full_like(gp[-1], p_b[-1])) and np.array_equal(grho[:, 0, :], np.repeat(rho_b[:, None], n, 1))
    e = np.array(errs)
    r = e[1] / e[2]
    assert np.all(r > 3.3) and np.all(r < 4.8), (e, r)


def _curl(Bx, By, Bz, h):
    """central-difference curl on the nodes [1:-1]^3 (numpy, test-side)."""
    hx, hy, hz = h
    d = lambda a, ax, hh: (np.roll(a, -1, ax) - np.roll(a, 1, ax))[1:-1, 1:-1, 1:-1] / (2 * hh)
    return (d(Bz, 1, hy) - d(By, 0, hz), d(Bx, 0, hz) - d(Bz, 2, hx), d(By, 2, hx) - d(Bx, 1, hy))


def _solve_smooth(orc, n, alpha, a, kappa):
    L = (1.0, 1.0, 1.0)
    x = grid(n, 1.0)
    Bz0 = np.sin(np.pi * x)[:, None] * np.sin(np.pi * x)[None, :] + 0.5 * np.sin(np.pi * x)[:, None] * np.sin(2 * np.pi * x)[None, :]
    f = a * np.exp(-kappa * x)
    P0, _ = orc.solve_boundary(Bz0, L[:2], tol=1e-12, max_cycles=60)
    P = np.zeros((n, n, n)); P[0] = P0
    P, _ = orc.solve_interior(P, f, alpha, L, tol=1e-12, max_cycles=80)
    return P, f, L, Bz0


def test_P10_divB_current_ansatz_and_force_balance_are_second_order(orc):
    """With P solved by the oracle: div B, eq (4) mu0 j = alpha B + xi grad(Bz) x ez, and eq (1)
    j x B - grad p - rho g ez (mu0 j = curl B) all vanish like h^2 (rms over the nodes at least
    1/8 of the box away from every wall: B is SET to 0 on the walls (C13), so the differences taken
    next to them are not consistent and are left out).  A wrong sign of xi (reading C1), of alpha,
    or of any B component breaks the trend."""
    alpha, mu0, g = 1.0, 0.5, 1.0
    res = []
    for n in (17, 33, 65):
        P, f, L, _ = _solve_smooth(orc, n, alpha, 0.5, 3.0)
        h = [1.0 / (n - 1)] * 3
        z = grid(n, 1.0)
        p_b, rho_b = np.exp(-z), np.exp(-z)
        dfdz = -3.0 * f
        Bx, By, Bz, p, rho = orc.fields(P, f, alpha, L, p_b, rho_b, mu0=mu0, g=g, dfdz=dfdz)
        d = lambda a, ax: (np.roll(a, -1, ax) - np.roll(a, 1, ax))[1:-1, 1:-1, 1:-1] / (2 * h[0])
        div = d(Bx, 2) + d(By, 1) + d(Bz, 0)
        cx, cy, cz = _curl(Bx, By, Bz, h)
        xi = -f[1:-1, None, None]
        I = np.s_[1:-1, 1:-1, 1:-1]
        e4 = (cx - alpha * Bx[I] - xi * d(Bz, 1), cy - alpha * By[I] + xi * d(Bz, 2), cz - alpha * Bz[I])
        jx, jy, jz = cx / mu0, cy / mu0, cz / mu0
        fx = jy * Bz[I] - jz * By[I] - d(p, 2)
        fy = jz * Bx[I] - jx * Bz[I] - d(p, 1)
        fz = jx * By[I] - jy * Bx[I] - d(p, 0) - rho[I] * g
        m = (n - 1) // 8
        w = np.s_[m:-m, m:-m, m:-m]
        rms = lambda *a: np.sqrt(np.mean(sum(q[w] ** 2 for q in a)))
        res.append([rms(div), rms(*e4), rms(fx, fy, fz), rms(Bx[I], By[I], Bz[I])])
    r = np.array(res)
    ratio = r[1, :3] / r[2, :3]
    assert np.all(ratio > 3.4) and np.all(ratio < 4.3), (r, ratio)
    assert np.all(r[2, :3] < 2e-2 * r[2, 3])                         # and small relative to |B|


def test_P12_force_free_gives_background_exactly(orc):
    """xi = 0 => p = p_b and rho = rho_b (bit-exact)."""
    n = 17
    P, f, L, _ = _solve_smooth(orc, n, 0.4, 0.0, 0.0)
    z = grid(n, 1.0)
    p_b, rho_b = np.exp(-z), 0.5 * np.exp(-z)
    _, _, _, p, rho = orc.fields(P, np.zeros(n), 0.4, L, p_b, rho_b)
    assert np.array_equal(p, np.broadcast_to(p_b[:, None, None], p.shape))
    assert np.array_equal(rho, np.broadcast_to(rho_b[:, None, None], rho.shape))


def test_P14_potential_field_is_curl_free(orc):
    rms = []
    for n in (17, 33, 65):
        P, f, L, _ = _solve_smooth(orc, n, 0.0, 0.0, 0.0)
        z = grid(n, 1.0)
        Bx, By, Bz, _, _ = orc.fields(P, f, 0.0, L, np.exp(-z), np.exp(-z))
        c = _curl(Bx, By, Bz, [1.0 / (n - 1)] * 3)
        w = np.s_[2:-2, 2:-2, 2:-2]
        rms.append(np.sqrt(np.mean(sum(q[w] ** 2 for q in c))))
    assert rms[1] / rms[2] > 3.0 and rms[0] / rms[1] > 2.5, rms


def test_bottom_plane_Bz_reproduces_the_magnetogram(orc):
    """Bz(x,y,0) = -(dxx+dyy)P on the bottom plane returns the prescribed Bz0 to solver tolerance
    (closes the loop eq (11) -> eq (5); C13)."""
    w = inputs.config(0)
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly), tol=1e-12, max_cycles=60)
    P = np.zeros(w.shape); P[0] = P0
    _, _, Bz, _, _ = orc.fields(P, w.f, w.alpha, w.L, w.p_b, w.rho_b)
    assert np.abs(Bz[0, 1:-1, 1:-1] - w.Bz0[1:-1, 1:-1]).max() <= 1e-9


# ----------------------------------------------------------------------- P11, P13 ------------
def test_P11_cycle_count_independent_of_mesh_size(orc):
    """multigrid convergence rate independent of the mesh size."""
    cyc2 = []
    for n in (33, 65, 129):
        w = inputs.config(0, shrink=1)
        Bz0 = inputs.gaussian_patches(n, n, 1.0, 1.0, [1.0, -1.0], [0.1, 0.1], [0.4, 0.6], [0.5, 0.5])
        _, info = orc.solve_boundary(Bz0, (1.0, 1.0))
        cyc2.append(info["cycles"])
    assert max(cyc2) - min(cyc2) <= 1 and max(cyc2) <= 18, cyc2
    cyc3 = []
    for n in (17, 33, 65):
        Bz0 = inputs.gaussian_patches(n, n, 1.0, 1.0, [1.0, -1.0], [0.1, 0.1], [0.4, 0.6], [0.5, 0.5])
        P0, _ = orc.solve_boundary(Bz0, (1.0, 1.0))
        P = np.zeros((n, n, n)); P[0] = P0
        _, info = orc.solve_interior(P, np.zeros(n), 0.5, (1.0, 1.0, 1.0))
        cyc3.append(info["cycles"])
        h = info["history"]
        assert 0.2 < h[-1] / h[-2] < 0.45                            # asymptotic V(2,2) factor ~0.35
    assert max(cyc3) - min(cyc3) <= 2 and max(cyc3) <= 25, cyc3


def test_P13_linearity_and_bipole_antisymmetry(orc):
    w = inputs.config(0)
    Lxy = (w.Lx, w.Ly)
    P0, i0 = orc.solve_boundary(w.Bz0, Lxy)
    P0s, _ = orc.solve_boundary(-3.0 * w.Bz0, Lxy)
    assert np.abs(P0s + 3.0 * P0).max() <= 1e-15
    assert i0["cycles"] == 16 and abs(np.abs(P0).max() - 7.07e-3) < 2e-5   # survey-time probe values
    P = np.zeros(w.shape); P[0] = P0
    P, info = orc.solve_interior(P, w.f, w.alpha, w.L)
    assert info["cycles"] == 22
    assert np.abs(P + P[:, :, ::-1]).max() <= 1e-15                  # antisymmetric about x = 1/2
    assert np.abs(P - P[:, ::-1, :]).max() <= 1e-15                  # symmetric about y = 1/2
    # stop rule (C10): first k with r_k <= tol r0
    h = info["history"]
    assert h[-1] <= 1e-10 * info["r0"] < h[-2]
    # continuing cycle by cycle gives the same iterates as one call
    Q = np.zeros(w.shape); Q[0] = P0
    r0 = 0.0
    for k in range(3):
        Q, inf = orc.solve_interior(Q, w.f, w.alpha, w.L, max_cycles=1, r0=r0)
        r0 = inf["r0"]
        assert inf["history"][0] == h[k]
