"""Field-line integration (the field lines of the paper's Figs 1, 4, 5):
RK4 through the trilinearly interpolated nodal B.  Pins of oracle.fieldlines (-m "not gpu") and parity of mhs_fieldlines
with it (-m gpu).  The paper prints no field-line coordinates (figures only), so closed forms and invariants pin the oracle."""
import numpy as np
import pytest

from paper_1307_6720_b200 import inputs


def _grid(n, L):
    z, y, x = np.meshgrid(*[np.linspace(0.0, l, m) for m, l in zip(n[::-1], L[::-1])], indexing="ij")
    return x, y, z


def test_uniform_field_gives_straight_lines(orc):
    """B = const: x_n = x_0 + n h B/|B| to rounding; the line ends at the last point inside the box; dir = -1 runs the other
    way; a seed outside the box gives no points."""
    n, L = (9, 7, 5), (1.0, 2.0, 0.5)
    b = np.array([1.0, 2.0, -0.5])
    B = [np.full(n[::-1], v) for v in b]
    seeds = np.array([[0.2, 0.3, 0.4], [0.9, 1.9, 0.05], [1.5, 0.1, 0.1]])
    h = 0.01
    lines, npts = orc.fieldlines(*B, L, seeds, h, 1000, +1)
    t = b / np.linalg.norm(b)
    for s in range(2):
        m = npts[s]
        # exits through z = 0 (seed 0) / x = 1 or y = 2 (seed 1): count = 1 + floor(distance / h) to within the rounding of the last step
        dist = min((np.where(t > 0, np.array(L) - seeds[s], seeds[s]) / np.abs(t)))
        assert abs(m - (1 + int(np.floor(dist / h)))) <= 1 and m >= 2
        want = seeds[s][None, :] + h * np.arange(m)[:, None] * t[None, :]
        assert np.abs(lines[s, :m] - want).max() < 1e-13
        assert np.all(np.isnan(lines[s, m:]))
    assert npts[2] == 0
    back, nb = orc.fieldlines(*B, L, seeds[:1], h, 1000, -1)
    assert np.abs(back[0, :nb[0]] - (seeds[0][None, :] - h * np.arange(nb[0])[:, None] * t[None, :])).max() < 1e-13
    # max_points caps the line; the seed counts as a point
    _, n5 = orc.fieldlines(*B, L, seeds[:1], h, 5, +1)
    assert n5[0] == 5


def test_rigid_rotation_closes_its_circles(orc):
    """B = (-(y - yc), x - xc, 0) is linear, so trilinear interpolation is exact and the field lines are circles: the radius
    is kept to O(h^5) over a turn (ratio 32 per halving of h: measured 6.9e-7, 2.1e-8, 6.7e-10 for h = 0.08, 0.04, 0.02) and the
    angle advances by h / r per step to O(h^4) (ratio -> 16)."""
    n, L = (17, 17, 5), (2.0, 2.0, 1.0)
    x, y, z = _grid(n, L)
    Bx, By, Bz = -(y - 1.0), (x - 1.0), np.zeros_like(x)
    r0 = 0.6
    seeds = np.array([[1.0 + r0, 1.0, 0.37]])
    errs = []
    for h in (0.04, 0.02):
        nstep = int(round(2 * np.pi * r0 / h))
        lines, npts = orc.fieldlines(Bx, By, Bz, L, seeds, h, nstep + 1, +1)
        assert npts[0] == nstep + 1
        p = lines[0]
        rad = np.hypot(p[:, 0] - 1.0, p[:, 1] - 1.0)
        ang = np.unwrap(np.arctan2(p[:, 1] - 1.0, p[:, 0] - 1.0))
        assert np.all(p[:, 2] == 0.37)
        errs.append((np.abs(rad - r0).max(), np.abs(ang - h / r0 * np.arange(nstep + 1)).max()))
        assert np.all(np.diff(ang) > 0)                       # counter-clockwise for dir = +1
    assert errs[0][0] < 1e-7 and 25.0 < errs[0][0] / errs[1][0] < 40.0, errs
    assert errs[0][1] < 1e-6 and 10.0 < errs[0][1] / errs[1][1] < 20.0, errs


def test_flux_function_is_constant_along_a_line(orc):
    """A 2.5D field B = (d psi/dz, b0, -d psi/dx) with psi = sin(pi x / Lx) exp(-q z): psi is constant along every field line.
    The nodal B is exact, what varies psi along the computed line is the trilinear interpolation error, O(h_grid^2): the drift
    falls by ~4 per grid halving; a transposed component or index in the sampler is an O(1) drift.  dir = -1 from the end
    of a line comes back to its seed within the integration error."""
    L, q, b0 = (2.0, 1.0, 1.0), 1.3, 0.25
    drift = []
    for m in (17, 33, 65):
        n = (m, 9, m)
        x, y, z = _grid(n, L)
        psi = lambda x, z: np.sin(np.pi * x / L[0]) * np.exp(-q * z)
        Bx = -q * psi(x, z)
        By = np.full_like(x, b0)
        Bz = -(np.pi / L[0]) * np.cos(np.pi * x / L[0]) * np.exp(-q * z)
        seeds = np.array([[1.65, 0.05, 0.02], [1.4, 0.1, 0.03], [1.2, 0.02, 0.01]])   # (x > Lx/2: Bz > 0, the lines rise and arch over)
        lines, npts = orc.fieldlines(Bx, By, Bz, L, seeds, 0.01, 400, +1)
        d = 0.0
        for s in range(3):
            p = lines[s, :npts[s]]
            assert npts[s] > 30
            ps = psi(p[:, 0], p[:, 2])
            d = max(d, np.abs(ps - ps[0]).max() / ps[0])
            assert np.all(np.diff(p[:, 1]) > 0)               # By > 0 everywhere
        drift.append(d)
        if m == 33:
            end = lines[1, npts[1] - 1][None, :]
            back, nb = orc.fieldlines(Bx, By, Bz, L, end, 0.01, npts[1], -1)
            assert nb[0] == npts[1] and np.abs(back[0, nb[0] - 1] - seeds[1]).max() < 1e-6
    assert drift[0] / drift[1] > 3.0 and drift[1] / drift[2] > 3.0 and drift[2] < 2e-3, drift


def test_a_null_stops_the_line(orc):
    """|B| <= bmin at a stage ends the line there (a null); with B = 0 everywhere only the seed is kept."""
    n, L = (5, 5, 5), (1.0, 1.0, 1.0)
    Z = np.zeros(n)
    _, npts = orc.fieldlines(Z, Z, Z, L, [[0.5, 0.5, 0.5]], 0.05, 10, +1)
    assert npts[0] == 1
    x, y, z = _grid(n, L)
    # B = (0.5 - x, 0, 0): lines run at unit speed towards the plane x = 0.5, where B vanishes, and end once a stage sees
    # |B| <= bmin (with bmin below half a step they would hop back and forth across the null for ever)
    lines, npts = orc.fieldlines(0.5 - x, Z, Z, L, [[0.1, 0.5, 0.5]], 0.03, 100, +1, bmin=0.02)
    assert 10 < npts[0] < 16 and 0.44 < lines[0, npts[0] - 1, 0] <= 0.5


# ------------------------------------------------------------------ GPU parity --------------------
def _solve_case(B, orc, name, dtype):
    import torch
    w = {"small": lambda: inputs.small(), "cfg1_65": lambda: inputs.config(1, shrink=2),
         "paper_ff_129": lambda: inputs.paper_example("force_free", 129)}[name]()
    S = B.Solver.from_workload(w, dtype=dtype)
    S.solve_boundary(torch.as_tensor(w.Bz0, dtype=dtype, device="cuda").contiguous())
    S.solve_interior(w.tol if dtype == torch.float64 else 1e-6, 100)
    Bf, _, _ = S.fields(want=("B",))
    return w, S, Bf


def _seeds(w, n):
    """seeds just above the base spread over the middle of the plane, plus a few higher up and one outside the box"""
    rng = inputs.SplitMix64(inputs.SEED_BASE + 4242)
    s = np.stack([rng.uniform(0.2, 0.8, n) * w.Lx, rng.uniform(0.2, 0.8, n) * w.Ly, rng.uniform(0.01, 0.3, n) * w.Lz], axis=1)
    s[-1] = [1.5 * w.Lx, 0.5 * w.Ly, 0.5 * w.Lz]
    return s


@pytest.mark.gpu
@pytest.mark.parametrize("direction", [1, -1])
@pytest.mark.parametrize("name", ["small", "cfg1_65", "paper_ff_129"])
def test_fieldlines_parity_fp64(orc, name, direction):
    """fp64: the kernel evaluates the same fma-ordered formulas as the oracle, so every point of every line and every
    point count is equal BIT FOR BIT (the exit tests decide an integer: both sides take them in fp64)."""
    import torch
    from paper_1307_6720_b200 import binding as B
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    w, S, Bf = _solve_case(B, orc, name, torch.float64)
    with S:
        seeds = _seeds(w, 257)
        step = 0.25 * min(w.Lx / (w.nx - 1), w.Ly / (w.ny - 1), w.Lz / (w.nz - 1))
        maxp = 600
        lines, npts = S.fieldlines(Bf, torch.as_tensor(seeds, device="cuda"), step, maxp, direction, bmin=1e-12)
        Bh = Bf.cpu().numpy()
        lo, no = orc.fieldlines(Bh[0], Bh[1], Bh[2], w.L, seeds, step, maxp, direction, bmin=1e-12)
        npts = npts.cpu().numpy(); lines = lines.cpu().numpy()
        assert np.array_equal(npts, no)
        assert no[-1] == 0 and no[:-1].min() >= 1 and no.max() > 50
        for s in range(len(seeds)):
            assert np.array_equal(lines[s, :no[s]], lo[s, :no[s]]), s


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["small", "cfg1_65"])
def test_fieldlines_parity_fp32(orc, name):
    """fp32 context: positions and B are float; against the fp64 oracle run on the same (fp32-rounded) B the points agree to
    1e-4 of the box over the first 200 steps of every line that both sides carry that far."""
    import torch
    from paper_1307_6720_b200 import binding as B
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    w, S, Bf = _solve_case(B, orc, name, torch.float32)
    with S:
        seeds = _seeds(w, 65).astype(np.float32).astype(np.float64)
        step = 0.25 * min(w.Lx / (w.nx - 1), w.Ly / (w.ny - 1), w.Lz / (w.nz - 1))
        lines, npts = S.fieldlines(Bf, torch.as_tensor(seeds, dtype=torch.float32, device="cuda"), step, 200, 1, bmin=1e-6)
        Bh = Bf.cpu().double().numpy()
        lo, no = orc.fieldlines(Bh[0], Bh[1], Bh[2], w.L, seeds, step, 200, 1, bmin=1e-6)
        npts = npts.cpu().numpy(); lines = lines.cpu().double().numpy()
        assert npts[-1] == 0 and no[-1] == 0
        worst = 0.0
        for s in range(len(seeds) - 1):
            m = min(npts[s], no[s])
            assert abs(int(npts[s]) - int(no[s])) <= 2 or m >= 20, (s, npts[s], no[s])
            worst = max(worst, np.abs(lines[s, :m] - lo[s, :m]).max() / max(w.L))
        assert worst <= 1e-4, worst
