"""Non-zero Dirichlet data for P on the side and top faces ("In principle other elliptic
equations can be defined on the other boundaries").  CPU part: the oracle's generic driver takes the boundary nodes of P as
Dirichlet data (orc_solve3) -- pinned here for data that is NOT zero on the sides and the top, against discrete closed forms.
GPU part: mhs_set_wall_data against the oracle, per iterate, converged, and through mhs_fields."""
import numpy as np
import pytest

from paper_1307_6720_b200 import inputs


def _zero_interior(P):
    Q = P.copy()
    Q[1:-1, 1:-1, 1:-1] = 0.0
    return Q


def test_oracle_linear_potential_is_reproduced_from_its_boundary_values(orc):
    """alpha = 0: every second difference of a + b x + c y + d z is zero, so it solves the discrete eq 8 exactly for any f(z).
    A wall value entering the operator at a wrong node, with a wrong sign or not at all cannot return it."""
    nz, ny, nx = 9, 17, 9
    L = (1.0, 2.0, 0.5)
    z, y, x = np.meshgrid(np.linspace(0, L[2], nz), np.linspace(0, L[1], ny), np.linspace(0, L[0], nx), indexing="ij")
    P = 0.3 + 1.1 * x - 0.7 * y + 2.0 * z
    f = 0.6 * np.exp(-4.0 * np.linspace(0, L[2], nz))
    got, info = orc.solve_interior(_zero_interior(P), f, 0.0, L, tol=1e-13, max_cycles=60)
    assert np.abs(got - P).max() <= 1e-11 * np.abs(P).max()
    assert orc.resnorm3(P, None, 1.0 + f, 0.0, L) <= 1e-10
    # and the fields of it: Bz = 0, Bx = alpha c, By = -alpha b at every node that is not on a side or the top -- the nodes
    # next to the walls take the wall values of P through the central differences
    alpha = 0.8
    Bx, By, Bz, p, rho = orc.fields(P, f, alpha, L, np.exp(-np.linspace(0, L[2], nz)), np.exp(-np.linspace(0, L[2], nz)))
    inner = (slice(0, nz - 1), slice(1, ny - 1), slice(1, nx - 1))
    assert np.abs(Bz[inner]).max() <= 1e-10
    assert np.abs(Bx[inner] - alpha * (-0.7)).max() <= 1e-11 and np.abs(By[inner] + alpha * 1.1).max() <= 1e-11


def test_oracle_separable_solution_with_data_on_sides_and_top(orc):
    """P = exp(a x) sin(m pi y / Ly) Z_k with Z from the three-term recurrence that makes eq 8 hold plane by plane
    (c_k (lx + ly) Z_k + (Z_{k+1} - 2 Z_k + Z_{k-1}) / hz^2 + alpha^2 Z_k = 0): an exact discrete solution that is non-zero on
    both x-faces and on the top, for z-dependent f and alpha != 0."""
    nz, ny, nx = 9, 9, 17
    L = (1.0, 1.0, 0.5)
    hx, hy, hz = L[0] / (nx - 1), L[1] / (ny - 1), L[2] / (nz - 1)
    alpha, a, m = 0.7, 1.3, 1
    f = 0.5 * np.exp(-3.0 * np.linspace(0, L[2], nz))
    lx = (np.exp(a * hx) - 2.0 + np.exp(-a * hx)) / hx**2                    # D_xx exp(a x) = lx exp(a x)
    ly = (2.0 * np.cos(m * np.pi * hy / L[1]) - 2.0) / hy**2                 # D_yy sin = ly sin
    Z = np.zeros(nz); Z[0], Z[1] = 1.0, 0.9
    for k in range(1, nz - 1):
        Z[k + 1] = 2.0 * Z[k] - Z[k - 1] - hz**2 * ((1.0 + f[k]) * (lx + ly) + alpha**2) * Z[k]
    X = np.exp(a * np.linspace(0, L[0], nx)); Y = np.sin(m * np.pi * np.linspace(0, L[1], ny) / L[1])
    P = Z[:, None, None] * Y[None, :, None] * X[None, None, :]
    assert abs(Z[-1]) > 0.05 and abs(X[0] - X[-1]) > 1.0                     # data on the top and on both x-faces
    assert orc.resnorm3(P, None, 1.0 + f, alpha, L) <= 1e-9 * np.abs(P).max() / hz**2
    got, info = orc.solve_interior(_zero_interior(P), f, alpha, L, tol=1e-13, max_cycles=80)
    assert np.abs(got - P).max() <= 1e-10 * np.abs(P).max()
    # negative control: with the x-face data dropped the same solve lands somewhere else
    Q = _zero_interior(P); Q[:, :, 0] = 0.0; Q[:, :, -1] = 0.0
    other, _ = orc.solve_interior(Q, f, alpha, L, tol=1e-13, max_cycles=80)
    assert np.abs(other - P)[1:-1, 1:-1, 1:-1].max() > 1e-2 * np.abs(P).max()


def test_oracle_wall_data_is_linear_superposition(orc):
    """The solution depends linearly on (bottom data, wall data): P(bottom, wall) = P(bottom, 0) + P(0, wall)."""
    w = inputs.small()
    G = inputs.wall_data(w)
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly))
    def start(bottom, wall):
        P = np.zeros(w.shape)
        if wall: P[:] = G
        P[1:-1, 1:-1, 1:-1] = 0.0
        P[0, 1:-1, 1:-1] = P0[1:-1, 1:-1] if bottom else 0.0
        return P
    sol = {k: orc.solve_interior(start(*k), w.f, w.alpha, w.L, tol=1e-13, max_cycles=80)[0] for k in ((1, 1), (1, 0), (0, 1))}
    assert np.abs(sol[(1, 1)] - sol[(1, 0)] - sol[(0, 1)]).max() <= 1e-10 * np.abs(sol[(1, 1)]).max()
    assert np.abs(sol[(0, 1)]).max() > 0.1 * np.abs(G).max()
