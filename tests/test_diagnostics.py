"""Diagnostics |B|, j = curl B / mu0, |j| (eq 2; the quantities of Figs 2, 4-7).
Pins of oracle.diagnostics (-m "not gpu") and parity of mhs_diagnostics with it (-m gpu)."""
import numpy as np
import pytest

from paper_1307_6720_b200 import inputs


def _grid(n, L):
    z, y, x = np.meshgrid(*[np.linspace(0.0, l, m) for m, l in zip(n[::-1], L[::-1])], indexing="ij")
    return x, y, z


def test_curl_of_a_linear_field_is_exact(orc):
    """B = (2z - 3y, 5x + z, 4y - x): curl B = (4 - 1, 2 + 1, 5 + 3) = (3, 3, 8) -- central and one-sided second-order
    differences are exact for linear fields, so j = curl B / mu0 to rounding at every node that is not a side / top wall,
    bottom plane included; on those walls j = 0; |B| is the Euclidean norm everywhere."""
    n, L, mu0 = (9, 7, 6), (1.0, 2.0, 0.5), 0.25
    x, y, z = _grid(n, L)
    Bx, By, Bz = 2 * z - 3 * y, 5 * x + z, 4 * y - x
    aB, jx, jy, jz, aJ = orc.diagnostics(Bx, By, Bz, L, mu0=mu0)
    assert np.allclose(aB, np.sqrt(Bx ** 2 + By ** 2 + Bz ** 2), rtol=1e-15)
    I = np.s_[:-1, 1:-1, 1:-1]
    for j, v in ((jx, 3.0), (jy, 3.0), (jz, 8.0)):
        assert np.abs(j[I] - v / mu0).max() < 1e-11
    assert np.abs(aJ[I] - np.sqrt(82.0) / mu0).max() < 1e-11
    for j in (jx, jy, jz, aJ):
        assert np.all(j[-1] == 0) and np.all(j[:, 0] == 0) and np.all(j[:, -1] == 0) and np.all(j[:, :, 0] == 0) and np.all(j[:, :, -1] == 0)


def test_curl_of_a_smooth_field_is_second_order(orc):
    """A field with every mixed derivative non-zero against its analytic curl: error ratio -> 4 per halving, in the interior
    and on the bottom plane (one-sided z differences); a transposed index or a wrong sign anywhere is an O(1) error."""
    L, mu0 = (1.0, 1.3, 0.8), 0.5
    errs = []
    for m in (17, 33, 65):
        x, y, z = _grid((m, m, m), L)
        Bx = np.sin(2 * y) * np.cos(3 * z) + x * z
        By = np.cos(x) * np.exp(z) + y * y
        Bz = np.sin(x + 2 * y) * (1 + z)
        cx = 2 * np.cos(x + 2 * y) * (1 + z) - np.cos(x) * np.exp(z)            # dy Bz - dz By
        cy = -3 * np.sin(2 * y) * np.sin(3 * z) + x - np.cos(x + 2 * y) * (1 + z)  # dz Bx - dx Bz
        cz = -np.sin(x) * np.exp(z) - 2 * np.cos(2 * y) * np.cos(3 * z)          # dx By - dy Bx
        aB, jx, jy, jz, aJ = orc.diagnostics(Bx, By, Bz, L, mu0=mu0)
        I = np.s_[:-1, 1:-1, 1:-1]
        errs.append(max(np.abs(j[I] - c[I] / mu0).max() for j, c in ((jx, cx), (jy, cy), (jz, cz))))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5, errs


def test_current_of_a_computed_equilibrium(orc):
    """On the oracle's own solution of a smooth problem, eq (4): mu0 j = alpha B + xi grad(Bz) x ez holds to O(h^2) away from
    the walls -- and for xi = 0 the current is parallel to the field, |j| = alpha |B| / mu0."""
    import importlib
    pins = importlib.import_module("test_oracle_pins")
    alpha, mu0 = 1.0, 0.5
    res = []
    for n in (17, 33, 65):
        P, f, L, _ = pins._solve_smooth(orc, n, alpha, 0.0, 0.0)
        z = np.linspace(0.0, 1.0, n)
        Bx, By, Bz, p, rho = orc.fields(P, f, alpha, L, np.exp(-z), np.exp(-z), mu0=mu0)
        aB, jx, jy, jz, aJ = orc.diagnostics(Bx, By, Bz, L, mu0=mu0)
        m = (n - 1) // 8
        w = np.s_[m:-m, m:-m, m:-m]
        res.append([np.sqrt(np.mean((mu0 * aJ[w] - alpha * aB[w]) ** 2)), np.sqrt(np.mean(aB[w] ** 2))])
    r = np.array(res)
    assert 3.3 < r[1, 0] / r[2, 0] < 4.5, r
    assert r[2, 0] < 2e-2 * r[2, 1]


@pytest.mark.gpu
@pytest.mark.parametrize("dtype_name", ["f64", "f32"])
@pytest.mark.parametrize("name", ["ragged", "cfg1_65", "paper_ff_129"])
def test_diagnostics_parity(orc, name, dtype_name):
    import torch
    from paper_1307_6720_b200 import binding as B
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    dt = torch.float64 if dtype_name == "f64" else torch.float32
    w = {"ragged": lambda: inputs.small(), "cfg1_65": lambda: inputs.config(1, shrink=2),
         "paper_ff_129": lambda: inputs.paper_example("force_free", 129)}[name]()
    with B.Solver.from_workload(w, dtype=dt) as S:
        S.solve_boundary(torch.as_tensor(w.Bz0, dtype=dt, device="cuda"))
        S.solve_interior(1e-6 if dt == torch.float32 else w.tol, w.max_cycles)
        Bf, _, _ = S.fields(want=("B",))
        aB, J, aJ = S.diagnostics(Bf)
        Bh = Bf.cpu().double().numpy()
        ref = orc.diagnostics(Bh[0], Bh[1], Bh[2], w.L, mu0=w.mu0)
        tol = 1e-12 if dt == torch.float64 else 2e-4     # fp32: first differences of fp32 data, eps / h
        sJ = np.abs(ref[4]).max()
        assert np.abs(aB.cpu().double().numpy() - ref[0]).max() <= (1e-14 if dt == torch.float64 else 1e-6) * np.abs(ref[0]).max()
        for q in range(3):
            assert np.abs(J[q].cpu().double().numpy() - ref[1 + q]).max() <= tol * sJ, q
        assert np.abs(aJ.cpu().double().numpy() - ref[4]).max() <= tol * sJ
        # subsets of outputs
        aB2, J2, aJ2 = S.diagnostics(Bf, want=("absJ",))
        assert aB2 is None and J2 is None and torch.equal(aJ2, aJ)
