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


# ====================================================================== GPU parity ======================
def _B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1307_6720_b200 import binding
    binding.lib()
    return binding, torch


def _dev(a, dtype):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda").contiguous()


def _host(t):
    return t.detach().cpu().double().numpy()


def _relmax(a, b):
    s = np.abs(b).max()
    return np.abs(a - b).max() / (s if s > 0 else 1.0)


def _aniso(n=65):
    """1 - xi from 0.05 at the base to 0.65 at the top (the regime of the paper's xi_2) on the config-1 sources."""
    w = inputs.config(1, shrink=128 // (n - 1))
    w.f = -(0.95 * np.exp(-1.0 * np.linspace(0.0, w.Lz, w.nz)))
    w.name = "aniso%d" % n
    return w


VW = {
    "ragged_17x33x9": lambda: inputs.small(),
    "cfg0_33": lambda: inputs.config(0),
    "cfg1_65": lambda: inputs.config(1, shrink=2),
    "aniso_65": lambda: _aniso(65),
    "cfg1_129": lambda: inputs.config(1),
    "cfg4_129x129x33": lambda: inputs.config(4, shrink=8),
}


@pytest.mark.gpu
@pytest.mark.parametrize("dtype_name", ["f64", "f32"])
@pytest.mark.parametrize("sweeps", [(2, 2), (1, 1), (2, 1)])
@pytest.mark.parametrize("name", ["ragged_17x33x9", "cfg0_33", "aniso_65", "cfg4_129x129x33"])
def test_zline_per_iterate_parity(orc, name, sweeps, dtype_name):
    """mhs_options.smoother = MHS_SMOOTH_ZLINE: single sweeps (levels 0 and 1, with a right-hand side on level 1) and eight
    V-cycle iterates against the oracle, 1e-12 (fp64) / 1e-5 (fp32) per iterate."""
    B, torch = _B()
    dtype = torch.float64 if dtype_name == "f64" else torch.float32
    tol = 1e-12 if dtype_name == "f64" else 1e-5
    optol = 1e-13 if dtype_name == "f64" else 2e-6
    w = VW[name]()
    a, b = sweeps
    c = 1.0 + w.f
    omega = 0.8
    with B.Solver.from_workload(w, dtype=dtype, n_pre=a, n_post=b, omega=omega, smoother=B.MHS_SMOOTH_ZLINE,
                                boundary_tol=1e-10 if dtype_name == "f64" else 1e-6) as S:
        if sweeps == (2, 2):
            for lvl in (0, 1):
                shp = S._shape(3, lvl)
                u = inputs.random_field(shp, 700 + lvl)
                rhs = None
                if lvl == 0:
                    u[0] = inputs.random_field(shp[1:], 710)
                else:
                    rhs = inputs.random_field(shp, 720)
                    S.level_set(3, lvl, 1, _dev(rhs, dtype))
                S.level_set(3, lvl, 0, _dev(u, dtype))
                S.op_smooth(3, lvl, 1)
                Ll = w.L
                ref = orc.zline3(u, rhs, c[:: 2**lvl], w.alpha, omega, Ll)
                assert _relmax(_host(S.level_get(3, lvl, 0)), ref) <= 4 * optol, lvl
        S.solve_boundary(_dev(w.Bz0, dtype))
        P = _host(S.get_potential())
        r0 = orc.resnorm3(P, None, c, w.alpha, w.L)
        for k in range(8):
            info = S.solve_interior(0.0, 1)
            P = orc.vcycle3s(P, None, c, w.alpha, w.L, omega=omega, n_pre=a, n_post=b, smoother=1)
            err = _relmax(_host(S.get_potential()), P)
            assert err <= tol, (name, sweeps, k, err)
            rk = orc.resnorm3(P, None, c, w.alpha, w.L)
            if rk / r0 > (1e-4 if dtype_name == "f32" else 1e-8):
                assert abs(info["history"][0] - rk) <= (1e-2 if dtype_name == "f32" else 1e-6) * rk


@pytest.mark.gpu
def test_zline_solve_to_tolerance_and_cycle_savings(orc):
    """One call to 1e-10 with z-line smoothing on the strongly anisotropic problem: the oracle's cycle count and solution,
    three times fewer cycles than point Jacobi needs on the same problem."""
    B, torch = _B()
    w = _aniso(65)
    with B.Solver.from_workload(w, omega=0.8, smoother=B.MHS_SMOOTH_ZLINE) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        P0 = _host(S.get_potential())
        iz = S.solve_interior(1e-10, 200)
        Po, oi = orc.solve_interior_opt(P0, w.f, w.alpha, w.L, omega=0.8, smoother=1, tol=1e-10, max_cycles=200)
        assert iz["converged"] and iz["cycles"] == oi["cycles"]
        assert _relmax(_host(S.get_potential()), Po) <= 1e-12
    with B.Solver.from_workload(w) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        ip = S.solve_interior(1e-10, 200)
        assert ip["converged"] and ip["cycles"] >= 3 * iz["cycles"], (ip["cycles"], iz["cycles"])


@pytest.mark.gpu
@pytest.mark.parametrize("flags", [0, 8])
@pytest.mark.parametrize("smoother,nfmg", [(0, 1), (0, 2), (1, 1)])
@pytest.mark.parametrize("name", ["ragged_17x33x9", "cfg0_33", "cfg1_65", "cfg1_129", "cfg4_129x129x33"])
def test_fmg_start_parity(orc, name, smoother, nfmg, flags):
    """mhs_options.fmg_cycles: (i) the full-multigrid iterate itself (a call whose tolerance it meets returns 0 cycles),
    (ii) the solve to tolerance -- r0, cycle count, solution -- against orc_solve_interior_opt."""
    B, torch = _B()
    w = VW[name]()
    omega = 0.8 if smoother else w.omega
    kw = dict(omega=omega, smoother=smoother, fmg_cycles=nfmg, flags=flags, dtype=torch.float64)
    with B.Solver.from_workload(w, **kw) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        P0 = _host(S.get_potential())
        i0 = S.solve_interior(1e30, 5)                      # any iterate meets this tolerance: FMG start only
        assert i0["cycles"] == 0 and i0["converged"]
        guess = orc.fmg_interior(P0, w.f, w.alpha, w.L, omega=omega, n_pre=w.n_pre, n_post=w.n_post, smoother=smoother, n_fmg=nfmg)
        assert _relmax(_host(S.get_potential()), guess) <= 1e-12
        c = 1.0 + w.f
        assert abs(i0["r0"] - orc.resnorm3(P0, None, c, w.alpha, w.L)) <= 1e-9 * i0["r0"]
        assert abs(i0["r_final"] - orc.resnorm3(guess, None, c, w.alpha, w.L)) <= 1e-6 * i0["r_final"]
        # a second call continues from the FMG iterate with ordinary cycles (no second FMG start)
        i1 = S.solve_interior(0.0, 1)
        P1 = orc.vcycle3s(guess, None, c, w.alpha, w.L, omega=omega, n_pre=w.n_pre, n_post=w.n_post, smoother=smoother)
        assert i1["cycles"] == 1 and _relmax(_host(S.get_potential()), P1) <= 1e-12
    with B.Solver.from_workload(w, **kw) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        info = S.solve_interior(w.tol, 100)
        Po, oi = orc.solve_interior_opt(P0, w.f, w.alpha, w.L, omega=omega, n_pre=w.n_pre, n_post=w.n_post, smoother=smoother,
                                        fmg=nfmg, tol=w.tol)
        assert info["converged"] and info["cycles"] == oi["cycles"], (info["cycles"], oi["cycles"])
        assert abs(info["r0"] - oi["r0"]) <= 1e-9 * oi["r0"]
        assert _relmax(_host(S.get_potential()), Po) <= 1e-12
        # mhs_set_potential is continued from, never replaced by an FMG start
        S.set_potential(_dev(P0, torch.float64))
        i2 = S.solve_interior(0.0, 1)
        P2 = orc.vcycle3s(P0, None, 1.0 + w.f, w.alpha, w.L, omega=omega, n_pre=w.n_pre, n_post=w.n_post, smoother=smoother)
        assert _relmax(_host(S.get_potential()), P2) <= 1e-12


@pytest.mark.gpu
def test_fmg_saves_cycles_at_full_size(orc):
    """BASELINE configs[2] (257^3): with a one-cycle-per-level FMG start the solve to 1e-10 needs fewer finest-level cycles
    and reaches the same potential; the FMG iterate is checked against the oracle (~1.5 V-cycles of oracle work)."""
    B, torch = _B()
    w = inputs.config(2)
    with B.Solver.from_workload(w) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        P0 = _host(S.get_potential())
        ia = S.solve_interior(w.tol, 100)
        Pa = S.get_potential().clone()
    with B.Solver.from_workload(w, fmg_cycles=1) as S:
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        i0 = S.solve_interior(1e30, 1)
        guess = orc.fmg_interior(P0, w.f, w.alpha, w.L)
        assert i0["cycles"] == 0 and _relmax(_host(S.get_potential()), guess) <= 1e-12
        S.solve_boundary(_dev(w.Bz0, torch.float64))
        ib = S.solve_interior(w.tol, 100)
        assert ib["converged"] and ib["cycles"] <= ia["cycles"] - 3, (ia["cycles"], ib["cycles"])
        assert abs(ib["r0"] - ia["r0"]) <= 1e-12 * ia["r0"]
        assert float((S.get_potential() - Pa).abs().max()) <= 1e-8 * float(Pa.abs().max())


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg0_33", "ragged_17x33x9", "cfg1_65"])
def test_jacobi_weight_option_parity(orc, name):
    """omega = 6/7 (the 3D smoothing-optimal Jacobi weight; C4 makes omega an option) through every kernel family."""
    B, torch = _B()
    w = VW[name]()
    om = 6.0 / 7.0
    for flags in (0, 8, 1):
        with B.Solver.from_workload(w, omega=om, flags=flags) as S:
            S.solve_boundary(_dev(w.Bz0, torch.float64))
            P = _host(S.get_potential())
            c = 1.0 + w.f
            for k in range(5):
                S.solve_interior(0.0, 1)
                P = orc.vcycle3(P, None, c, w.alpha, w.L, omega=om, n_pre=w.n_pre, n_post=w.n_post)
                assert _relmax(_host(S.get_potential()), P) <= 1e-12, (flags, k)


@pytest.mark.gpu
def test_solve_batch_equals_member_by_member(orc):
    """mhs_solve_batch on three magnetograms of one region: every member equals, bit for bit, what the separate calls give,
    and the oracle's solve of that member; infos carry each member's cycle count."""
    B, torch = _B()
    ws = [inputs.config(1, shrink=2, replica=r) for r in range(3)]
    w = ws[0]
    bz = torch.stack([_dev(x.Bz0, torch.float64) for x in ws])
    with B.Solver.from_workload(w) as S:
        out, infos = S.solve_batch(bz, w.tol, 100, want=("P", "B", "rho"))
        for b, x in enumerate(ws):
            S.solve_boundary(_dev(x.Bz0, torch.float64))
            i = S.solve_interior(w.tol, 100)
            assert i["cycles"] == infos[b]["cycles"] and infos[b]["converged"]
            assert torch.equal(S.get_potential(), out["P"][b])
            Bf, _, rho = S.fields(want=("B", "rho"))
            assert torch.equal(Bf, out["B"][b]) and torch.equal(rho, out["rho"][b])
            P0, _ = orc.solve_boundary(x.Bz0, (w.Lx, w.Ly))
            Po = np.zeros(w.shape); Po[0] = P0
            Po, oi = orc.solve_interior(Po, w.f, w.alpha, w.L)
            assert oi["cycles"] == infos[b]["cycles"] and _relmax(_host(out["P"][b]), Po) <= 1e-12
        # max_cycles too small for every member: reported, results are the valid 2nd iterates
        out2, infos2 = S.solve_batch(bz, w.tol, 2, want=("P",))
        assert all(i["cycles"] == 2 and not i["converged"] for i in infos2)
        empty, none = S.solve_batch(bz[:0], w.tol, 5)
        assert none == [] and empty["P"].shape[0] == 0
