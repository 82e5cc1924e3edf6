"""Pins of the CPU oracle (oracle/nanobte_ref.c) against things that are NOT the oracle:
dense LAPACK solves assembled independently in tests/fvgeom.py (P1, P2), a closed-form
discrete slab solution (P3), exact invariants (P4, P5, P8), the plain/synthetic fixed point
(P6) and the classical radiative-equilibrium slab (P7).  CPU only (`-m "not gpu"`).

Citations: PAPER.md:55 (Eq. 4), 59 (Eq. 5), 62 (Eq. 6), 71 (Eq. 7), 77-97 (Eq. 8-12), 91 (Eq. 11),
104/110 (transport matrix I/tau + v K_i), 133-137 (diffusive: linear profile; ballistic: wall jumps).
"""
import numpy as np
import pytest

import fvgeom
from oracle.ref import RefSolver, OracleError
from paper_2607_03226_b200 import workloads as wl

TH, DF, SP, MX = wl.THERMALIZING, wl.DIFFUSE, wl.SPECULAR, wl.MIXED


def small_bands(B, seed=0, lo=-12.5, hi=-10.5):
    """B bands with dx/Lambda of order 0.1..10 on ~10 nm cells (so that no term of the update is negligible).
    Synthetic-mode tests use lo=-11.3 (dx/Lambda < 1): the synthetic iteration is only stable for optically
    thin cells (reading R14f)."""
    rng = np.random.default_rng(seed)
    return {"C": rng.uniform(0.5e6, 2e6, B), "v": rng.uniform(3e3, 7e3, B), "tau": 10.0 ** rng.uniform(lo, hi, B)}


def tiny_problems():
    out = {}
    tags = [(TH, 303.0), (TH, 298.5), (DF, 0.0), (SP, 0.0), (MX, 0.0)]
    rng = np.random.default_rng(7)
    # 2-D 4x4, non-uniform spacing, left therm / right mixed / bottom diffuse / top specular
    out["quad4x4"] = wl.make_structured_problem(
        4, 4, 1, rng.uniform(5e-9, 15e-9, 4), rng.uniform(5e-9, 15e-9, 4), np.ones(1), small_bands(2, 1),
        wl.inplane_quadrature(8), tags, [0, 4, 2, 3, 0, 0], Qdot=rng.uniform(0, 1e17, 16), p_seed=11)
    # 3-D 3x3x3, all four kinds
    out["hex3x3x3"] = wl.make_structured_problem(
        3, 3, 3, rng.uniform(5e-9, 15e-9, 3), rng.uniform(5e-9, 15e-9, 3), rng.uniform(5e-9, 15e-9, 3),
        small_bands(2, 2), wl.product_quadrature(2, 4), tags, [0, 1, 2, 4, 3, 4], Qdot=rng.uniform(0, 1e17, 27),
        p_seed=12)
    # masked L-shape 4x3x3 (re-entrant corner: cells with several boundary faces)
    act = np.ones((3, 3, 4), bool)
    act[1:, 1:, 2:] = False
    out["Lshape4x3x3"] = wl.make_structured_problem(
        4, 3, 3, 8e-9, 9e-9, 10e-9, small_bands(3, 3), wl.product_quadrature(2, 4), tags, [0, 4, 2, 4, 3, 4],
        active=act, Qdot=rng.uniform(0, 1e17, 36) * act.ravel(), p_seed=13)
    # jittered triangles 4x4x2 with a (one-quad) hole, therm / therm / specular / diffuse hole
    tri = wl.config_triangles(n=4, side=40e-9, B=2, D=8, hole_radius=6e-9, jitter=0.2, seed=3)
    tri["bands"] = small_bands(2, 4)
    tri["Qdot"] = rng.uniform(0, 1e17, tri["mesh"]["n_cells"])
    out["tri4x4"] = tri
    return out


TINY = tiny_problems()


def random_T(problem, seed):
    rng = np.random.default_rng(seed)
    m = problem["mesh"]
    n = m["n_cells"] if problem["kind"] == "unstructured" else m["nx"] * m["ny"] * m["nz"]
    return problem["T_ref"] + rng.uniform(-2.0, 2.0, n)


# ------------------------------------------------------------------------------------------------
# P1: one sweep == dense LAPACK solve of (I/tau_b + v_b K_i) eps = rhs
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
def test_P1_sweep_equals_dense_solve(name):
    pr = TINY[name]
    g = fvgeom.Geom(pr)
    r = RefSolver(pr, T_init=random_T(pr, 5))
    for _ in range(2):  # make eps^n and the diffuse averages non-trivial
        r.sweep()
        r.update_temperature()
    eps_prev = g.to_active(r.get_e())
    theta = g.to_active(r.get_T(0)) - pr["T_ref"]
    r.sweep()
    got = g.to_active(r.get_e())
    want = g.dense_sweep(theta, eps_prev)
    assert np.abs(want).max() > 0
    for b in range(got.shape[0]):
        assert np.abs(got[b] - want[b]).max() <= 1e-12 * np.abs(want[b]).max()
    # boundary values used by the sweep, and the moments that follow it
    bcv, G = g.boundary_values(eps_prev, pr["T_ref"])
    np.testing.assert_allclose(r.get_boundary_values(), bcv, rtol=1e-13, atol=1e-13 * np.abs(bcv).max())
    r.update_temperature()
    th_SI, th_en, q = g.moments(want)
    np.testing.assert_allclose(g.to_active(r.get_T(0)) - pr["T_ref"], th_SI, rtol=0, atol=1e-12 * np.abs(th_SI).max())
    np.testing.assert_allclose(g.to_active(r.get_T(1)) - pr["T_ref"], th_en, rtol=0, atol=1e-12 * np.abs(th_en).max())
    qa = r.get_q()[g.act2cell]
    np.testing.assert_allclose(qa, q[:, :g.dim], rtol=0, atol=1e-12 * np.abs(q).max())
    _, G2 = g.boundary_values(want, pr["T_ref"])
    np.testing.assert_allclose(r.get_G(), G2, rtol=0, atol=1e-12 * np.abs(G2).max())


# ------------------------------------------------------------------------------------------------
# P2: converged iteration == one global direct solve of the coupled (eps, theta) system
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
@pytest.mark.parametrize("mode", ["plain", "synthetic"])
def test_P2_global_fixed_point_tiny(name, mode):
    pr = dict(TINY[name])
    if mode == "synthetic":
        pr["bands"] = small_bands(len(pr["bands"]["C"]), 21, lo=-11.3)
    g = fvgeom.Geom(pr)
    eps_fp, th_fp = g.fixed_point()
    r = RefSolver(pr)
    res = r.solve(1e-12, 20000, mode)
    assert res["converged"], res
    th = g.to_active(r.get_T(0)) - pr["T_ref"]
    assert np.abs(th - th_fp).max() <= 2e-10 * max(1.0, np.abs(th_fp).max())
    eps = g.to_active(r.get_e())
    for b in range(eps.shape[0]):
        assert np.abs(eps[b] - eps_fp[b]).max() <= 1e-8 * np.abs(eps_fp[b]).max()


def test_P2_global_fixed_point_config0():
    """BASELINE.json configs[0] itself (6,400 + 400 unknowns) is pinned by the direct solve."""
    pr = wl.config_gray_square()
    g = fvgeom.Geom(pr)
    eps_fp, th_fp = g.fixed_point()
    r = RefSolver(pr)
    res = r.solve(pr["tol"], pr["max_iter"], "plain")
    assert res["converged"] and res["iters"] == 35  # R9/R11: count includes the satisfying iteration
    th = r.get_T(0) - 300.0
    # stopping at |dT| < 1e-10 leaves an error of that order times 1/(1 - rho)
    assert np.abs(th - th_fp).max() < 5e-10
    # P8 symmetry, exact to rounding
    T = r.get_T(0).reshape(20, 20)
    assert np.abs(T - T[::-1, :]).max() < 1e-12
    assert np.abs((T - 300.0) + (T[:, ::-1] - 300.0)).max() < 1e-12
    # energy: no source -> heat in through the hot wall = heat out through the cold wall, diffuse walls ~0
    H = r.get_boundary_heat()
    assert abs(H[0] + H[1]) < 1e-9 * abs(H[0]) and abs(H[2]) < 1e-9 * abs(H[0])
    assert H[0] < 0 < H[1]  # outward positive: hot wall injects


# ------------------------------------------------------------------------------------------------
# P3: closed-form discrete slab (gray, 4 half-offset in-plane directions, specular side walls)
# ------------------------------------------------------------------------------------------------
def slab_problem(nx, ny, L, kn, Th=301.0, Tc=299.0, C=1.66e6, v=6400.0):
    lam = kn * L
    bands = {"C": np.array([C]), "v": np.array([v]), "tau": np.array([lam / v])}
    tags = [(TH, Th), (TH, Tc), (SP, 0.0)]
    pr = wl.make_structured_problem(nx, ny, 1, L / nx, L / nx, 1.0, bands, wl.inplane_quadrature(4), tags,
                                    [0, 1, 2, 2, 0, 0], T_ref=0.5 * (Th + Tc))
    return pr, lam


@pytest.mark.parametrize("nx,ny,kn", [(8, 3, 0.05), (8, 3, 1.0), (16, 2, 30.0), (5, 1, 0.3), (40, 1, 0.02)])
def test_P3_closed_form_discrete_slab(nx, ny, kn):
    L, Th, Tc, C, v = 100e-9, 301.0, 299.0, 1.66e6, 6400.0
    pr, lam = slab_problem(nx, ny, L, kn, Th, Tc, C, v)
    r = RefSolver(pr)
    res = r.solve(1e-13, 200000, "plain")
    assert res["converged"]
    sx = 1.0 / np.sqrt(2.0)
    a = lam * sx / (L / nx)
    dT = Th - Tc
    J = dT * (1 + 2 * a) / (1 + 2 * a + nx)
    i = np.arange(1, nx + 1)
    T_exact = Th - J / 2 - (2 * i - 1) * J / (2 * (1 + 2 * a))
    T = r.get_T(0).reshape(ny, nx)
    assert np.abs(T - T_exact[None, :]).max() < 5e-11
    q = r.get_q().reshape(ny, nx, 2)
    qx = C * v * sx * a * J / (1 + 2 * a)
    np.testing.assert_allclose(q[..., 0], qx, rtol=1e-9)
    assert np.abs(q[..., 1]).max() < 1e-9 * qx
    H = r.get_boundary_heat()
    face_flux = C * v * sx * J / 2  # W/m^2, times wall length ny*h (unit depth)
    np.testing.assert_allclose(H[1], face_flux * ny * (L / nx), rtol=1e-9)
    np.testing.assert_allclose(H[0], -H[1], rtol=1e-9)


def test_P3_limits_ballistic_jump_and_fourier_profile():
    """north_star checks 2 and 3: Kn >> 1 -> flat interior at the mean wall temperature, wall
    jump dT/2; Kn << 1 -> linear Fourier profile between the walls and q = -kappa dT/dx."""
    L, Th, Tc = 100e-9, 301.0, 299.0
    pr, _ = slab_problem(10, 1, L, 1e4, Th, Tc)
    r = RefSolver(pr)
    assert r.solve(1e-13, 1000)["converged"]
    T = r.get_T(0)
    assert np.abs(T - 300.0).max() < 2e-3  # O(1/Kn)
    assert abs((Th - T[0]) - 1.0) < 2e-3  # jump = dT/2
    # Fourier flux needs dx << lambda: the upwind scheme's effective MFP is lambda + dx/(2|s_x|)
    nx = 400
    pr, lam = slab_problem(nx, 1, L, 0.02, Th, Tc)  # dx/lambda = 0.125
    r = RefSolver(pr)
    assert r.solve(1e-12, 100000, "synthetic")["converged"]
    T, q = r.get_T(0), r.get_q()[:, 0]
    x = (np.arange(nx) + 0.5) * L / nx
    slope, icpt = np.polyfit(x, T, 1)
    assert np.abs(T - (slope * x + icpt)).max() < 1e-9  # exactly linear (closed form P3: T_i linear in i)
    assert abs(icpt - Th) < 0.05 and abs(slope * L + (Th - Tc)) < 0.08  # walls nearly without jump
    assert r.kappa == pytest.approx(1.66e6 * 6400.0 * lam / 2, rel=1e-12)  # C v Lambda / 2 in-plane (R14d)
    lam_eff = lam + (L / nx) / (2 / np.sqrt(2.0)) * 1.0  # first-order upwind numerical diffusion, |s_x| = 1/sqrt2
    # cell-centre moment q (Eq. 7) is exactly Fourier's -kappa dT/dx on this profile; the conserved FACE flux
    # carries the numerical diffusion (closed form P3: face flux = q_cell (1 + 1/(2a)))
    assert q[nx // 2] == pytest.approx(-r.kappa * slope, rel=1e-6)
    assert r.get_boundary_heat()[1] / (L / nx) == pytest.approx(-r.kappa * slope * lam_eff / lam, rel=1e-6)


# ------------------------------------------------------------------------------------------------
# P4: isothermal preservation
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
def test_P4_isothermal(name):
    pr = dict(TINY[name])
    m = dict(pr["mesh"])
    m["tags"] = [(t, 300.0) for (t, _) in m["tags"]]
    pr["mesh"] = m
    pr["Qdot"] = np.zeros_like(pr["Qdot"])
    pr["T_ref"] = 300.0
    for T_ref in (300.0, 250.0):  # deviational zero, and a non-zero uniform deviation
        pr["T_ref"] = T_ref
        r = RefSolver(pr, T_init=np.full(len(pr["Qdot"]), 300.0))
        # a uniform deviation must be carried by the reflecting-wall caches too, so start them consistently
        if T_ref == 300.0:
            for _ in range(3):
                r.sweep()
                d = r.update_temperature()
            assert d == 0.0
        else:  # eps^0 = 0 is NOT the isothermal state about another T_ref: the iteration must find 300 K again
            assert r.solve(1e-12, 200000)["converged"]
        g = fvgeom.Geom(pr)
        assert np.abs(g.to_active(r.get_T(0)) - 300.0).max() < 1e-9
    r = RefSolver(pr | {"T_ref": 300.0})
    res = r.solve(1e-10, 10)
    assert res["iters"] == 1 and res["last_dT"] == 0.0
    assert np.abs(r.get_e()).max() == 0.0


# ------------------------------------------------------------------------------------------------
# P5: per-cell energy balance after EVERY sweep, global balance, source split
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
def test_P5_cell_energy_balance_every_sweep(name):
    pr = TINY[name]
    g = fvgeom.Geom(pr)
    r = RefSolver(pr, T_init=random_T(pr, 9))
    beta = (pr["bands"]["C"] / pr["bands"]["tau"]).sum()
    Q = np.asarray(pr["Qdot"])[g.act2cell]
    for it in range(6):
        th_old = g.to_active(r.get_T(0)) - pr["T_ref"]
        r.sweep()
        r.update_temperature()
        eps = g.to_active(r.get_e())
        th_SI = g.to_active(r.get_T(2)) - pr["T_ref"]
        res, scale = g.cell_balance_residual(eps, r.get_boundary_values(), th_SI, th_old)
        assert (np.abs(res) <= 1e-12 * scale).all(), (it, np.abs(res / scale).max())
        # global: boundary heat = generation - beta-term (exact at any iteration)
        H = r.get_boundary_heat().sum()
        want = (g.vol * Q).sum() - beta * (g.vol * (th_SI - th_old)).sum()
        assert abs(H - want) <= 1e-11 * scale.sum()


def test_P5_converged_boundary_heat_equals_generation():
    """north_star check 4: net boundary heat = integrated generation to 1e-10 relative (after converging
    well below the solve tolerance)."""
    pr = wl.config_nongray_square(n=12, side=1e-6 * 12 / 128, B=3, D=8, sigma=20e-9, peak=1e18)
    pr["bands"] = small_bands(3, 5)
    r = RefSolver(pr)
    assert r.solve(1e-14, 20000)["converged"]
    g = fvgeom.Geom(pr)
    gen = (g.vol * pr["Qdot"]).sum()
    assert r.get_boundary_heat().sum() == pytest.approx(gen, rel=1e-10)


# ------------------------------------------------------------------------------------------------
# P6: synthetic mode reaches the plain fixed point (and its CG solves the dense diffusion system)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
def test_P6_diffusion_correction_is_dense_solve(name):
    pr = TINY[name]
    g = fvgeom.Geom(pr)
    r = RefSolver(pr, T_init=random_T(pr, 3))
    th_old = g.to_active(r.get_T(0)) - pr["T_ref"]
    r.sweep()
    r.update_temperature()
    th_SI = g.to_active(r.get_T(2)) - pr["T_ref"]
    it, _ = r.diffusion_correct()
    beta = (pr["bands"]["C"] / pr["bands"]["tau"]).sum()
    # R14d in closed form: unit direction vectors spanning the mesh's own dimension give the kinetic-theory value
    # kappa = (1/dim) sum_b C_b v_b^2 tau_b whatever the quadrature (1/3 C v Lambda in 3-D, 1/2 in-plane)
    kappa = (pr["bands"]["C"] * pr["bands"]["v"] ** 2 * pr["bands"]["tau"]).sum() / g.dim
    assert r.kappa == pytest.approx(kappa, rel=1e-13)
    M = g.diffusion_matrix(kappa)
    assert np.abs(M - M.T).max() <= 1e-12 * np.abs(M).max()
    leak = g.reflecting_leak(g.to_active(r.get_e()), r.get_boundary_values())
    assert np.abs(leak).max() > 0
    delta = np.linalg.solve(M, g.vol * beta * (th_SI - th_old) + leak)
    got = g.to_active(r.get_T(0)) - pr["T_ref"] - th_SI
    assert np.abs(got - delta).max() <= 1e-9 * np.abs(delta).max()
    assert 0 < it <= g.n_act + 5


# ------------------------------------------------------------------------------------------------
# P9: Fourier initial guess (O9, reading R21)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(TINY))
def test_P9_fourier_guess_is_dense_conduction_solve(name):
    """theta^0 against a dense LAPACK solve of the conduction problem assembled here from the raw face geometry
    (fvgeom): interior two-point fluxes, Dirichlet T_w at thermalizing faces at the centre-to-face distance, zero flux
    elsewhere, source V Qdot -- and the integral balance: what leaves through the thermalizing faces is what is generated."""
    pr = TINY[name]
    g = fvgeom.Geom(pr)
    if not (g.bf_type == 0).any():
        pytest.skip("no thermalizing face")
    kappa = (pr["bands"]["C"] * pr["bands"]["v"] ** 2 * pr["bands"]["tau"]).sum() / g.dim
    M = g.diffusion_matrix(kappa)
    Q = np.zeros(g.n_act) if pr.get("Qdot") is None else g.to_active(np.asarray(pr["Qdot"], dtype=float))
    rhs = g.vol * Q
    out = 0.0
    for (a, nbr, bf, A, n, d) in g.faces:
        if bf >= 0 and g.bf_type[bf] == 0:
            rhs[a] += kappa * A / d * (g.bf_Tw[bf] - pr["T_ref"])
    th = np.linalg.solve(M, rhs)
    r = RefSolver(pr, T_init=random_T(pr, 4))  # whatever theta was before, the guess replaces it
    it = r.init_fourier()
    got = g.to_active(r.get_T(0)) - pr["T_ref"]
    scale = max(np.abs(th).max(), 1e-300)
    assert np.abs(got - th).max() <= 1e-9 * scale
    assert 0 < it <= g.n_act + 5
    for (a, nbr, bf, A, n, d) in g.faces:
        if bf >= 0 and g.bf_type[bf] == 0:
            out += kappa * A / d * (got[a] - (g.bf_Tw[bf] - pr["T_ref"]))
    gen = (g.vol * Q).sum()
    assert out == pytest.approx(gen, rel=1e-8, abs=1e-9 * kappa * np.abs(got).max() * g.bf_area.max() / max(np.sqrt(g.vol.max()), 1e-300))


def test_P9_fourier_guess_closed_forms():
    """Slab between thermalizing walls at x = 0 and x = L, reflecting elsewhere, uniform cells of size h.
    (a) no source: the two-point-flux solution is the straight line through the wall temperatures, exactly, at the cell
    centres.  (b) uniform source, both walls at T_ref: theta_i = Q/(2 kappa) x_i (L - x_i) + Q h^2/(8 kappa): the second
    difference of a quadratic is exact, and the half-cell wall distance shifts the parabola by a constant
    (both checked to rounding)."""
    n, L = 16, 200e-9
    pr = wl.config_gray_square(n=n, D=8)
    h = L / n
    xc = (np.arange(n) + 0.5) * h
    kappa = (pr["bands"]["C"] * pr["bands"]["v"] ** 2 * pr["bands"]["tau"]).sum() / 2
    r = RefSolver(pr)
    r.init_fourier()
    th = (r.get_T(0) - pr["T_ref"]).reshape(n, n)
    line = 1.0 + (-1.0 - 1.0) * xc / L       # walls at 301 K and 299 K, T_ref 300 K
    assert np.abs(th - line[None, :]).max() <= 1e-12
    pr2 = dict(pr)
    m2 = dict(pr["mesh"])
    m2["tags"] = [(t[0], 300.0) if t[0] == 0 else t for t in pr["mesh"]["tags"]]
    pr2["mesh"] = m2
    Q = 1e17
    pr2["Qdot"] = np.full(n * n, Q)
    r2 = RefSolver(pr2)
    r2.init_fourier()
    th2 = (r2.get_T(0) - pr2["T_ref"]).reshape(n, n)
    para = Q / (2 * kappa) * xc * (L - xc) + Q * h * h / (8 * kappa)
    assert np.abs(th2 - para[None, :]).max() <= 1e-10 * para.max()


def test_P9_fourier_start_reaches_the_same_fixed_point():
    """The guess changes the iterate path, not the fixed point: solve() from theta^0 ends at the converged field of the
    run from T_ref (to the tolerance of the two runs), in fewer iterations on a diffusive case."""
    pr = wl.config_gray_square(n=12, D=8)
    pr["bands"] = dict(pr["bands"])
    pr["bands"]["tau"] = pr["bands"]["tau"] * 0.05  # Kn = 0.025: diffusive, where the Fourier field is close
    a, b = RefSolver(pr), RefSolver(pr)
    ra = a.solve(1e-10, 20000)
    b.init_fourier()
    rb = b.solve(1e-10, 20000)
    assert ra["converged"] and rb["converged"]
    assert np.abs(a.get_T(0) - b.get_T(0)).max() <= 1e-7
    assert rb["iters"] < ra["iters"]


def test_P6_plain_equals_synthetic_config0_family():
    # the paper's use case is the diffusive side; cells stay optically thin (R14f)
    for n, kn_scale in ((12, 1.0), (24, 0.1)):
        pr = wl.config_gray_square(n=n, D=8)
        pr["bands"]["tau"] = pr["bands"]["tau"] * kn_scale
        a, b = RefSolver(pr), RefSolver(pr)
        ra, rb = a.solve(1e-11, 50000, "plain"), b.solve(1e-11, 50000, "synthetic")
        assert ra["converged"] and rb["converged"]
        assert np.abs(a.get_T(0) - b.get_T(0)).max() < 1e-8
        if kn_scale < 0.5:
            assert 5 * rb["iters"] < ra["iters"]  # acceleration where it is meant to help


# ------------------------------------------------------------------------------------------------
# P7: continuous-limit anchor -- radiative-equilibrium gray slab (integral equation, solved here)
# ------------------------------------------------------------------------------------------------
def radiative_slab(tauL, n=2000):
    """phi(t) = 0.5 [E2(t) + int_0^tauL phi(t') E1(|t-t'|) dt'] for black walls at phi=1 (t=0), 0 (t=tauL);
    piecewise-constant collocation with the exact cell integrals of E1 (via E2).  Returns
    (Psi = q / (C v dT / 4), hot-wall jump / dT)."""
    from scipy.special import expn
    h = tauL / n
    t = (np.arange(n) + 0.5) * h
    edges = np.arange(n + 1) * h
    # int_{a}^{b} E1(|t - t'|) dt' = E2(|t-b|) ... signs handled per side
    d_lo = t[:, None] - edges[None, :-1]
    d_hi = t[:, None] - edges[None, 1:]
    K = np.where(d_hi >= 0, expn(2, np.abs(d_hi)) - expn(2, np.abs(d_lo)),
                 np.where(d_lo <= 0, expn(2, np.abs(d_lo)) - expn(2, np.abs(d_hi)),
                          2.0 - expn(2, np.abs(d_lo)) - expn(2, np.abs(d_hi))))
    phi = np.linalg.solve(np.eye(n) - 0.5 * K, 0.5 * expn(2, t))
    # net flux at t = 0 (constant through the slab): Psi = 2 [E3(0) - int phi E2 dt'] = 1 - 2 sum_j phi_j [E3]_j
    Psi = 1.0 - 2.0 * (phi * (expn(3, edges[:-1]) - expn(3, edges[1:]))).sum()
    # wall jump: 1 - phi(0+), linear extrapolation of the two first collocation values
    jump = 1.0 - (1.5 * phi[0] - 0.5 * phi[1])
    return Psi, jump, t / tauL, phi


@pytest.mark.slow
@pytest.mark.parametrize("tauL", [0.1, 1.0, 5.0])
def test_P7_radiative_slab_anchor(tauL):
    Psi, jump, xs, phi = radiative_slab(tauL)
    # textbook end points of this classical problem: Psi -> 1 as tauL -> 0, Psi ~ (4/3)/(tauL + 1.42) when thick
    assert 0 < Psi < 1
    if tauL >= 5:
        assert Psi == pytest.approx((4 / 3) / (tauL + 1.4209), rel=0.01)
    L, nx, C, v = 100e-9, 256, 1.66e6, 6400.0
    lam = L / tauL
    bands = {"C": np.array([C]), "v": np.array([v]), "tau": np.array([lam / v])}
    tags = [(TH, 301.0), (TH, 299.0), (SP, 0.0)]
    quad = wl.product_quadrature(16, 4, polar_axis=0)  # polar axis = slab normal
    pr = wl.make_structured_problem(nx, 1, 1, L / nx, L / nx, 1.0, bands, quad, tags, [0, 1, 2, 2, 0, 0])
    r = RefSolver(pr)
    assert r.solve(1e-11, 20000, "plain")["converged"]
    T = r.get_T(0)
    q = r.get_q()[nx // 2, 0]
    assert q / (C * v * 2.0 / 4) == pytest.approx(Psi, rel=0.015)
    # first-cell temperature against the integral-equation profile at the same position
    phi_at = np.interp((np.arange(nx) + 0.5) / nx, xs, phi)
    assert np.abs((T - 299.0) / 2.0 - phi_at).max() < 0.01


# ------------------------------------------------------------------------------------------------
# structured == unstructured on identical cells; error paths
# ------------------------------------------------------------------------------------------------
def test_structured_and_polygon_paths_agree():
    tags = [(TH, 302.0), (TH, 299.0), (DF, 0.0), (SP, 0.0)]
    bands, quad = small_bands(2, 8), wl.inplane_quadrature(8)
    ps = wl.make_structured_problem(5, 4, 1, 7e-9, 9e-9, 1.0, bands, quad, tags, [0, 1, 2, 3, 0, 0])
    pu = dict(ps)
    pu["kind"] = "unstructured"
    pu["mesh"] = wl.quads_as_unstructured(5, 4, 7e-9, 9e-9, lambda side: [0, 1, 2, 3][side], tags)
    a, b = RefSolver(ps), RefSolver(pu)
    for _ in range(5):
        a.sweep(); b.sweep()
        a.update_temperature(); b.update_temperature()
    assert np.abs(a.get_e() - b.get_e()).max() <= 1e-12 * np.abs(a.get_e()).max()
    np.testing.assert_allclose(a.get_T(0), b.get_T(0), rtol=0, atol=1e-12)


def test_error_paths():
    pr = wl.config_gray_square(n=4, D=8)
    bad = dict(pr); bad["mesh"] = dict(pr["mesh"]); bad["mesh"]["bf_cell"] = pr["mesh"]["bf_cell"][:-1]
    bad["mesh"]["bf_side"] = pr["mesh"]["bf_side"][:-1]; bad["mesh"]["bf_tag"] = pr["mesh"]["bf_tag"][:-1]
    with pytest.raises(OracleError) as e:
        RefSolver(bad)
    assert e.value.code == -5
    # specular wall whose mirror direction is missing from the quadrature
    q = wl.inplane_quadrature(8)
    q = {"s": q["s"][[0, 1, 2, 3, 4, 5, 6]], "w": q["w"][[0, 1, 2, 3, 4, 5, 6]], "dim": 2}
    sp = wl.config_gray_square(n=4, D=8, wall=SP); sp["quad"] = q
    with pytest.raises(OracleError) as e:
        RefSolver(sp)
    assert e.value.code in (-6, -8)
    # all-reflecting box cannot run the synthetic step
    tags = [(SP, 0.0)]
    box = wl.make_structured_problem(3, 3, 1, 1e-8, 1e-8, 1.0, small_bands(1), wl.inplane_quadrature(4), tags,
                                     [0, 0, 0, 0, 0, 0])
    r = RefSolver(box)
    with pytest.raises(OracleError) as e:
        r.solve(1e-9, 5, "synthetic")
    assert e.value.code == -9


def test_golden_config0_file_matches_oracle_and_fixed_point():
    """tests/golden/config0_oracle.txt is what the committed script wrote from oracle/ only, and is itself within the
    stopping error of the dense fixed point (P2): a stored value that both the oracle and the GPU tests answer to."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config0_oracle.txt")
    lines = open(path).read().splitlines()
    iters = int([ln for ln in lines if ln.startswith("# iterations")][0].split()[-1])
    T = np.array([[float(x) for x in ln.split()] for ln in lines if not ln.startswith("#")]).reshape(-1)
    pr = wl.config_gray_square()
    r = RefSolver(pr)
    res = r.solve(pr["tol"], pr["max_iter"])
    assert res["iters"] == iters == 35
    assert np.abs(r.get_T(0) - T).max() < 1e-12
    _, th_fp = fvgeom.Geom(pr).fixed_point()
    assert np.abs((T - 300.0) - th_fp).max() < 5e-10
