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


# ------------------------------------------------------------------------------------------------------------------
# GPU: mhs_set_wall_data against the oracle
# ------------------------------------------------------------------------------------------------------------------
def _gpu_case(w, dtype, flags, orc, iterates=3):
    import torch
    from paper_1307_6720_b200 import binding
    TOL = {torch.float64: 1e-12, torch.float32: 1e-5}[dtype]
    G = inputs.wall_data(w)
    if dtype == torch.float32:
        G = G.astype(np.float32).astype(np.float64)          # both sides take the data the GPU can hold
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda")
    rel = lambda a, b: np.abs(a - b).max() / np.abs(b).max()
    with binding.Solver.from_workload(w, dtype=dtype, flags=flags, bc=(binding.MHS_BC_DIRICHLET_DATA, binding.MHS_BC_DIRICHLET_DATA)) as S:
        S.solve_boundary(dev(w.Bz0))
        S.set_wall_data(dev(G))
        P0 = S.get_boundary().cpu().double().numpy()
        # the oracle's starting iterate: wall data on the sides and the top, the 2D solution on the bottom plane, zero inside
        Po = G.copy()
        Po[1:-1, 1:-1, 1:-1] = 0.0
        Po[0, 1:-1, 1:-1] = P0[1:-1, 1:-1]
        start = S.get_potential().cpu().double().numpy()
        assert rel(start, Po) <= 1e-15 if dtype == torch.float64 else rel(start, Po) <= 1e-7
        r0 = 0.0
        for it in range(iterates):                                     # per iterate (C21)
            info = S.solve_interior(1e-30, 1)
            Po, oi = orc.solve_interior(Po, w.f, w.alpha, w.L, omega=w.omega, n_pre=w.n_pre, n_post=w.n_post, tol=1e-30, max_cycles=1, r0=r0)
            r0 = oi["r0"]
            got = S.get_potential().cpu().double().numpy()
            assert rel(got, Po) <= TOL, (it, rel(got, Po))
            if it == 0:
                assert abs(info["r0"] - r0) <= 50 * TOL * r0
        # converged: restart from the 2D solution, solve to tolerance
        S.solve_boundary(dev(w.Bz0))
        tol = 1e-10 if dtype == torch.float64 else 1e-5
        info = S.solve_interior(tol, 80)
        Pc = G.copy(); Pc[1:-1, 1:-1, 1:-1] = 0.0; Pc[0, 1:-1, 1:-1] = P0[1:-1, 1:-1]
        Pc, oc = orc.solve_interior(Pc, w.f, w.alpha, w.L, omega=w.omega, n_pre=w.n_pre, n_post=w.n_post, tol=tol, max_cycles=80)
        got = S.get_potential().cpu().double().numpy()
        if dtype == torch.float64:
            assert info["cycles"] == oc["cycles"]
        assert rel(got, Pc) <= (TOL if dtype == torch.float64 else 20 * TOL)
        assert np.abs(got[:, :, 0] - G[:, :, 0]).max() <= 1e-6 * np.abs(G).max() and np.abs(got[-1] - G[-1])[1:-1, 1:-1].max() <= 1e-6 * np.abs(G).max()
        # fields of the full potential (the nodes next to the walls see the wall values)
        Bf, p, rho = S.fields()
        ref = orc.fields(got, w.f, w.alpha, w.L, w.p_b, w.rho_b, mu0=w.mu0, g=w.g)
        FT = 1e-11 if dtype == torch.float64 else 2e-3
        bmax = max(np.abs(ref[q]).max() for q in range(3))
        for q in range(3):
            assert np.abs(Bf[q].cpu().double().numpy() - ref[q]).max() <= FT * bmax, q
        assert np.abs(p.cpu().double().numpy() - ref[3]).max() <= FT * np.abs(ref[3]).max()
        if dtype == torch.float64:
            assert np.abs(rho.cpu().double().numpy() - ref[4]).max() <= 1e-10 * np.abs(ref[4]).max()
        return info


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["small_cluster", "cfg1_65_mid", "cfg1_65_big", "cfg1_65_big_sep", "small_ref"])
@pytest.mark.parametrize("f32", [False, True])
def test_wall_data_parity(orc, case, f32):
    import torch
    from paper_1307_6720_b200 import binding
    w = inputs.small() if case.startswith("small") else inputs.config(1, shrink=2)
    flags = {"small_cluster": 0, "cfg1_65_mid": 0, "cfg1_65_big": binding.MHS_FLAG_BIG_LEVEL_KERNELS,
             "cfg1_65_big_sep": binding.MHS_FLAG_BIG_LEVEL_KERNELS | binding.MHS_FLAG_SEPARATE_PROLONG,
             "small_ref": binding.MHS_FLAG_REFERENCE_KERNELS}[case]
    _gpu_case(w, torch.float32 if f32 else torch.float64, flags, orc)


@pytest.mark.gpu
def test_wall_data_state_and_zero_data(orc):
    """Without mhs_set_wall_data (or with zeros) a wall context returns what an ordinary context returns; the call is refused
    on an ordinary context; one face may stay MHS_BC_DIRICHLET_ZERO."""
    import torch
    from paper_1307_6720_b200 import binding
    w = inputs.small()
    bz = torch.as_tensor(w.Bz0, device="cuda")
    with binding.Solver.from_workload(w) as S:
        S.solve_boundary(bz); S.solve_interior(1e-10, 60)
        Pz = S.get_potential().cpu().numpy()
        with pytest.raises(binding.MHSError) as e:
            S.set_wall_data(torch.zeros(w.shape, dtype=torch.float64, device="cuda"))
        assert e.value.status == binding.MHS_ERR_STATE
    with binding.Solver.from_workload(w, bc=(1, 1)) as S:
        S.solve_boundary(bz); S.solve_interior(1e-10, 60)
        assert np.abs(S.get_potential().cpu().numpy() - Pz).max() <= 1e-12 * np.abs(Pz).max()
    G = inputs.wall_data(w)
    with binding.Solver.from_workload(w, bc=(0, 1)) as S:            # data on the top only: the side values of G are ignored
        S.solve_boundary(bz); S.set_wall_data(torch.as_tensor(G, device="cuda")); S.solve_interior(1e-10, 80)
        got = S.get_potential().cpu().numpy()
    Po = np.zeros(w.shape); Po[-1, 1:-1, 1:-1] = G[-1, 1:-1, 1:-1]
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly)); Po[0] = P0
    Po, _ = orc.solve_interior(Po, w.f, w.alpha, w.L, tol=1e-10, max_cycles=80)
    assert np.abs(got - Po).max() <= 1e-12 * np.abs(Po).max()
    with pytest.raises(binding.MHSError):
        binding.Solver.from_workload(w, bc=(1, 1), smoother=binding.MHS_SMOOTH_ZLINE if hasattr(binding, "MHS_SMOOTH_ZLINE") else 1)


@pytest.mark.gpu
def test_wall_data_from_elliptic_problems_on_the_other_faces(orc):
    """PAPER.md:96 as a whole: "other elliptic equations ... on the other boundaries".  A Poisson problem (eq 11's kind) is
    solved on the top face and on the two x-faces by boundary-only contexts (nz = 1), their solutions become the wall data of
    the 3D solve; the oracle does the same with its 2D and 3D drivers.  Every face problem has P = 0 on its own edges, so the
    faces agree along the edges of the box."""
    import torch
    from paper_1307_6720_b200 import binding
    w = inputs.config(1, shrink=4)                                           # 33^3
    nz, ny, nx = w.shape
    rng = inputs.SplitMix64(inputs.SEED_BASE + 777)
    faces = {"top": (nx, ny, w.Lx, w.Ly), "x0": (ny, nz, w.Ly, w.Lz), "x1": (ny, nz, w.Ly, w.Lz)}
    G = np.zeros(w.shape)
    Go = np.zeros(w.shape)
    for name, (n1, n2, L1, L2) in faces.items():
        src = inputs.random_patches(rng, 2, n1, n2, L1, L2, 0.1 * L1, 0.25 * L1)
        with binding.Solver(n1, n2, 1, L=(L1, L2, 1.0)) as F:
            F.solve_boundary(torch.as_tensor(src, device="cuda"))
            sol = F.get_boundary().cpu().numpy()
        solo, _ = orc.solve_boundary(src, (L1, L2))
        assert np.abs(sol - solo).max() <= 1e-12 * np.abs(solo).max()
        for arr, s in ((G, sol), (Go, solo)):
            if name == "top": arr[nz - 1] = s
            elif name == "x0": arr[:, :, 0] = s
            else: arr[:, :, nx - 1] = s
    with binding.Solver.from_workload(w, bc=(1, 1)) as S:
        S.solve_boundary(torch.as_tensor(w.Bz0, device="cuda"))
        S.set_wall_data(torch.as_tensor(G, device="cuda"))
        info = S.solve_interior(1e-10, 80)
        got = S.get_potential().cpu().numpy()
    P0, _ = orc.solve_boundary(w.Bz0, (w.Lx, w.Ly))
    Po = Go.copy(); Po[1:-1, 1:-1, 1:-1] = 0.0; Po[0, 1:-1, 1:-1] = P0[1:-1, 1:-1]
    Po, oi = orc.solve_interior(Po, w.f, w.alpha, w.L, tol=1e-10, max_cycles=80)
    assert info["cycles"] == oi["cycles"]
    assert np.abs(got - Po).max() <= 1e-12 * np.abs(Po).max()
    assert np.abs(got[nz - 1]).max() > 0 and np.abs(got[:, :, 0]).max() > 0


@pytest.mark.gpu
def test_wall_data_full_size_first_iterates(orc):
    """BASELINE configs[2] at full size (257^3 fp64, default flags) with wall data: the finest level then runs the temporally
    blocked smoother in its right-hand-side variants (with the norm by-product, with the prolongation folded in) and the
    separable restriction with a right-hand side, in the launch shapes of the big grid.  Two iterates against the oracle."""
    import torch
    from paper_1307_6720_b200 import binding
    w = inputs.config(2)
    G = inputs.wall_data(w, amp=0.05)
    with binding.Solver.from_workload(w, bc=(1, 1)) as S:
        S.solve_boundary(torch.as_tensor(w.Bz0, device="cuda"))
        S.set_wall_data(torch.as_tensor(G, device="cuda"))
        P0 = S.get_boundary().cpu().numpy()
        Po = G.copy(); Po[1:-1, 1:-1, 1:-1] = 0.0; Po[0, 1:-1, 1:-1] = P0[1:-1, 1:-1]
        r0 = 0.0
        for it in range(2):
            S.solve_interior(1e-30, 1)
            Po, oi = orc.solve_interior(Po, w.f, w.alpha, w.L, omega=w.omega, n_pre=w.n_pre, n_post=w.n_post, tol=1e-30, max_cycles=1, r0=r0)
            r0 = oi["r0"]
            got = S.get_potential().cpu().numpy()
            assert np.abs(got - Po).max() <= 1e-12 * np.abs(Po).max(), it
        assert S.profile()["sweeps_l0"] > 0
