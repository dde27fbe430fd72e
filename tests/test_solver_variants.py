"""Solver variants inside "a multigrid method": z-line Jacobi smoothing for strong
(1 - xi) anisotropy, a full-multigrid start, other Jacobi weights, batches of magnetograms.  They change the iterates, so each
has its own oracle function; this file pins those (-m "not gpu") and checks the CUDA path against them (-m gpu)."""
import numpy as np
import pytest

from paper_1307_6720_b200 import inputs
from test_oracle_pins import (T1, R1, kron3, interior, sinmode, lam, grid, _dense_level)

W23 = 2.0 / 3.0


def _dense_T(nx, ny, nz, hx, hy, hz, c, alpha):
    """The z-line part of L on the interior unknowns: diagonal of L + the two z-neighbours."""
    mx, my, mz = nx - 2, ny - 2, nz - 2
    A = _dense_level(nx, ny, nz, hx, hy, hz, c, alpha)
    offz = (np.diag(np.ones(mz - 1), 1) + np.diag(np.ones(mz - 1), -1)) / hz**2
    return np.diag(np.diag(A)) + kron3(offz, np.eye(my), np.eye(mx))


# ------------------------------------------------------------------ z-line Jacobi: pins ----------------
@pytest.mark.parametrize("dims,L", [((9, 7, 9), (1.0, 0.8, 1.1)), ((5, 9, 17), (0.5, 1.0, 2.0)), ((7, 5, 3), (1.0, 1.0, 0.3))])
def test_zline_equals_dense_formulation(orc, dims, L):
    """unew = u + omega T^-1 (rhs - L u) with dense L and T (variable c_k, non-zero Dirichlet data on the bottom plane, rhs)."""
    nx, ny, nz = dims
    h = [Lq / (n - 1) for Lq, n in zip(L, dims)]
    c = 1.0 + 0.9 * np.exp(-3.0 * grid(nz, L[2]))
    alpha, omega = 0.6, 0.85
    u = inputs.random_field((nz, ny, nx), 71)
    u[0] = inputs.random_field((ny, nx), 72)
    rhs = inputs.random_field((nz, ny, nx), 73)
    A = _dense_level(nx, ny, nz, *h, c, alpha)
    T = _dense_T(nx, ny, nz, *h, c, alpha)
    r = interior(orc.residual3(u, rhs, c, alpha, L)).ravel()       # (pinned on its own; carries the boundary data)
    want = interior(u).ravel() + omega * np.linalg.solve(T, r)
    got = orc.zline3(u, rhs, c, alpha, omega, L)
    assert np.abs(interior(got).ravel() - want).max() <= 1e-13 * np.abs(want).max()
    # boundary branch: every boundary node passes through
    mask = np.ones_like(u, dtype=bool); mask[1:-1, 1:-1, 1:-1] = False
    assert np.array_equal(got[mask], u[mask])
    # and T really is "L without the horizontal neighbours": A - T has zero diagonal and no z-coupling
    O = A - T
    assert np.abs(np.diag(O)).max() == 0.0


def test_zline_symbol_on_sine_modes(orc):
    """Constant c: a sine mode is multiplied by 1 - omega lambda_L / lambda_T, lambda_L = -c(lx+ly) - lz + alpha^2,
    lambda_T = D + (2/hz^2) cos(theta_z) = -2c/hx^2 - 2c/hy^2 - lz + alpha^2."""
    nx, ny, nz = 17, 33, 9
    L = (1.0, 2.0, 0.5)
    alpha, omega, cc = 0.7, 0.8, 1.3
    hx, hy, hz = [Lq / (n - 1) for Lq, n in zip(L, (nx, ny, nz))]
    c = np.full(nz, cc)
    for (a, b, d) in [(1, 1, 1), (3, 5, 2), (15, 31, 7), (8, 1, 4)]:
        u = sinmode(nz, d)[:, None, None] * sinmode(ny, b)[None, :, None] * sinmode(nx, a)[None, None, :]
        lx, ly, lz = lam(nx, L[0], a), lam(ny, L[1], b), lam(nz, L[2], d)
        lamL = -cc * (lx + ly) - lz + alpha**2
        lamT = -2 * cc / hx**2 - 2 * cc / hy**2 - lz + alpha**2
        np.testing.assert_allclose(orc.zline3(u, None, c, alpha, omega, L), (1.0 - omega * lamL / lamT) * u, rtol=0, atol=2e-14)


def test_zline_is_exact_without_horizontal_coupling_and_keeps_the_fixed_point(orc):
    """(i) On a domain so wide that c/hx^2, c/hy^2 are negligible L = T, and ONE sweep with omega = 1 solves every line:
    the residual drops by ten orders.  (ii) A solution of L u = rhs is a fixed point of the sweep for any omega."""
    nx, ny, nz = 9, 9, 33
    L = (1e5, 1e5, 1.0)
    c = 1.0 + 0.5 * np.exp(-4.0 * grid(nz, 1.0))
    rhs = inputs.random_field((nz, ny, nx), 74)
    u = np.zeros((nz, ny, nx)); u[0] = inputs.random_field((ny, nx), 75)
    r0 = orc.resnorm3(u, rhs, c, 0.3, L)
    u1 = orc.zline3(u, rhs, c, 0.3, 1.0, L)
    assert orc.resnorm3(u1, rhs, c, 0.3, L) <= 1e-9 * r0
    L2 = (1.0, 1.3, 0.7)
    us = orc.direct3(u, rhs, c, 0.3, L2)
    for om in (0.5, 1.0):
        assert np.abs(orc.zline3(us, rhs, c, 0.3, om, L2) - us).max() <= 1e-12 * np.abs(us).max()


def _dense_vcycle_s(level, dims, h, c, alpha, omega, n1, n2, v, rhs, orc, smoother):
    nx, ny, nz = dims
    A = _dense_level(nx, ny, nz, *h, c, alpha)
    if orc.is_coarsest(nx, ny, nz, level, 0):
        return np.linalg.solve(A, rhs)
    M = _dense_T(nx, ny, nz, *h, c, alpha) if smoother == 1 else np.diag(np.diag(A))
    for _ in range(n1):
        v = v + omega * np.linalg.solve(M, rhs - A @ v)
    R = kron3(R1(nz), R1(ny), R1(nx))
    cd = ((nx - 1) // 2 + 1, (ny - 1) // 2 + 1, (nz - 1) // 2 + 1)
    ec = _dense_vcycle_s(level + 1, cd, [2 * q for q in h], c[::2], alpha, omega, n1, n2, np.zeros(R.shape[0]), R @ (rhs - A @ v), orc, smoother)
    v = v + 8.0 * R.T @ ec
    for _ in range(n2):
        v = v + omega * np.linalg.solve(M, rhs - A @ v)
    return v


@pytest.mark.parametrize("smoother", [0, 1])
@pytest.mark.parametrize("dims,L", [((9, 9, 9), (1.0, 1.0, 1.0)), ((9, 9, 5), (1.0, 1.3, 0.4)), ((5, 9, 17), (0.5, 1.0, 1.5))])
def test_vcycle_with_smoother_option_equals_dense_matrix_formulation(orc, dims, L, smoother):
    """Every line of orc_vcycle3s, per iterate, against matrix products on tiny grids; smoother = 0 is orc_vcycle3 itself."""
    nx, ny, nz = dims
    h = [Lq / (n - 1) for Lq, n in zip(L, dims)]
    c = 1.0 + 0.7 * np.exp(-2.5 * grid(nz, L[2]))
    alpha = 0.8
    P = np.zeros((nz, ny, nx)); P[0] = inputs.random_field((ny, nx), 31)
    rhs_eff = np.zeros((nz - 2, ny - 2, nx - 2)); rhs_eff[0] = -P[0, 1:-1, 1:-1] / h[2] ** 2
    rhs_eff = rhs_eff.ravel()
    v = np.zeros_like(rhs_eff)
    exact = np.linalg.solve(_dense_level(nx, ny, nz, *h, c, alpha), rhs_eff)
    Q = P.copy()
    for it in range(5):
        P = orc.vcycle3s(P, None, c, alpha, L, omega=0.8, n_pre=2, n_post=1, smoother=smoother)
        v = _dense_vcycle_s(0, dims, h, c, alpha, 0.8, 2, 1, v, rhs_eff, orc, smoother)
        assert np.abs(interior(P).ravel() - v).max() <= 1e-13 * np.abs(exact).max(), it
        if smoother == 0:
            Q = orc.vcycle3(Q, None, c, alpha, L, omega=0.8, n_pre=2, n_post=1)
            assert np.array_equal(P, Q)


def test_zline_cures_the_strong_z_coupling_of_small_1_minus_xi(orc):
    """The reason for the option: with 1 - xi = 0.05 near the base the horizontal coupling is 20 times
    weaker than the vertical one, and point Jacobi V(2,2) cycles crawl; z-line Jacobi restores the textbook factor."""
    n = 33
    L = (1.0, 1.0, 1.0)
    z = grid(n, 1.0)
    f = -(0.95 * np.exp(-1.0 * z))                    # 1 - xi from 0.05 at the base to 0.65 at the top
    P = np.zeros((n, n, n)); P[0] = sinmode(n, 2)[:, None] * sinmode(n, 3)[None, :] + 0.3 * inputs.random_field((n, n), 5)
    _, ip = orc.solve_interior_opt(P, f, 0.5, L, smoother=0, tol=1e-10, max_cycles=200)
    _, iz = orc.solve_interior_opt(P, f, 0.5, L, smoother=1, omega=0.8, tol=1e-10, max_cycles=200)
    assert iz["cycles"] <= 14 and ip["cycles"] >= 3 * iz["cycles"], (ip["cycles"], iz["cycles"])
    # both converge to the same discrete solution
    Pp, _ = orc.solve_interior_opt(P, f, 0.5, L, smoother=0, tol=1e-12, max_cycles=400)
    Pz, _ = orc.solve_interior_opt(P, f, 0.5, L, smoother=1, omega=0.8, tol=1e-12, max_cycles=400)
    assert np.abs(Pp - Pz).max() <= 1e-9 * np.abs(Pp).max()


# ------------------------------------------------------------------ full-multigrid start: pins ----------
@pytest.mark.parametrize("smoother", [0, 1])
def test_fmg_equals_its_dense_matrix_formulation(orc, smoother):
    """orc_fmg_interior on 9 x 9 x 9 (three levels) restated with dense matrices: injection of the bottom data, exact coarsest
    solve, trilinear interpolation of the whole coarse solution (8 R^T on the interior + the bottom data's share), n_fmg
    V-cycles per level."""
    dims, L = (9, 9, 9), (1.0, 1.2, 0.9)
    nx, ny, nz = dims
    f = 0.6 * np.exp(-2.0 * grid(nz, L[2]))
    alpha, omega, n_fmg = 0.7, 0.8, 2
    P = np.zeros((nz, ny, nx)); P[0] = inputs.random_field((ny, nx), 91)
    got = orc.fmg_interior(P, f, alpha, L, omega=omega, n_pre=2, n_post=1, smoother=smoother, n_fmg=n_fmg)
    assert np.array_equal(got[0], P[0]) and np.all(got[-1] == 0)

    def level(l):
        s = 2**l
        d = tuple((m - 1) // s + 1 for m in dims)
        return d, [s * Lq / (m - 1) for Lq, m in zip(L, dims)], (1.0 + f)[::s], P[0][::s, ::s]

    def rhs_of(d, h, bottom):
        r = np.zeros((d[2] - 2, d[1] - 2, d[0] - 2)); r[0] = -bottom[1:-1, 1:-1] / h[2] ** 2
        return r.ravel()

    nl = 3
    assert orc.is_coarsest(3, 3, 3, 2, 0) and not orc.is_coarsest(5, 5, 5, 1, 0)
    d2, h2, c2, b2 = level(2)
    v = np.linalg.solve(_dense_level(*d2, *h2, c2, alpha), rhs_of(d2, h2, b2))
    for l in (1, 0):
        d, h, c, b = level(l)
        dc, hc, cc, bc = level(l + 1)
        # interpolate the coarse solution INCLUDING its bottom plane: embed, interpolate with the oracle's (pinned) operator
        Uc = np.zeros((dc[2], dc[1], dc[0])); Uc[0] = bc; Uc[1:-1, 1:-1, 1:-1] = v.reshape(dc[2] - 2, dc[1] - 2, dc[0] - 2)
        Uf = orc.prolong_add3(Uc, np.zeros((d[2], d[1], d[0])))
        v = interior(Uf).ravel()
        for _ in range(n_fmg):
            v = _dense_vcycle_s(l, d, h, c, alpha, omega, 2, 1, v, rhs_of(d, h, b), orc, smoother)
    assert np.abs(interior(got).ravel() - v).max() <= 1e-13 * np.abs(v).max()


def test_fmg_start_is_at_discretisation_accuracy_and_saves_cycles(orc):
    """What FMG is for: one V-cycle per level leaves an algebraic error of the order of the discretisation error, so the
    solve to 1e-10 (measured against the SAME r0, the zero-interior residual) needs fewer fine-grid cycles -- and lands on
    the same solution."""
    w = inputs.config(1, shrink=4)                                 # 33^3, f = 0.5 exp(-5 z)
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly))
    P = np.zeros(w.shape); P[0] = P0
    Pa, ia = orc.solve_interior_opt(P, w.f, w.alpha, w.L, fmg=0)
    Pb, ib = orc.solve_interior_opt(P, w.f, w.alpha, w.L, fmg=1)
    assert abs(ia["r0"] - ib["r0"]) <= 1e-12 * ia["r0"]
    assert ib["cycles"] <= ia["cycles"] - 3, (ia["cycles"], ib["cycles"])
    assert np.abs(Pa - Pb).max() <= 1e-8 * np.abs(Pa).max()
    guess = orc.fmg_interior(P, w.f, w.alpha, w.L)
    c = 1.0 + w.f
    assert orc.resnorm3(guess, None, c, w.alpha, w.L) <= 5e-2 * ia["r0"]          # (measured 3e-2: worth ~4 cycles)
    # fmg = 0 is orc_solve_interior itself
    Pc, ic = orc.solve_interior(P, w.f, w.alpha, w.L)
    assert ic["cycles"] == ia["cycles"] and np.array_equal(Pa, Pc)


def test_jacobi_weight_six_sevenths_is_the_better_3d_smoother(orc):
    """omega is an option (C4).  For the 7-point operator the smoothing-optimal Jacobi weight is 6/7 (2D: 4/5): with it a
    V(2,2) solve of a force-free problem needs no more cycles than with 2/3."""
    w = inputs.config(0)
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly))
    P = np.zeros(w.shape); P[0] = P0
    _, a = orc.solve_interior(P, w.f, w.alpha, w.L, omega=2.0 / 3.0)
    _, b = orc.solve_interior(P, w.f, w.alpha, w.L, omega=6.0 / 7.0)
    assert b["cycles"] <= a["cycles"]
