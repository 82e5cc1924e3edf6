"""Parity of the CUDA library (through its C ABI) against the CPU oracle, element by element, on the same seeded
inputs (`-m gpu`).  Bar (BASELINE.json north_star): per-sweep e_{b,s} and T within 1e-10 max-norm relative error
(deviational variables, per band -- SURVEY.md 8(d)), converged T within 1e-8 K with an identical iteration count.
"""
import numpy as np
import pytest

# max|dtheta| histories: the entries are differences of fields of size |theta| <= ~10 K, so two correct evaluations
# with different summation orders differ by a few tens of ulp(10 K) ~ 2e-15 each; 1e-13 is four orders below every
# convergence tolerance used here (R11) and far above that noise.
HIST_ATOL = 1e-13

from oracle.ref import RefSolver
from paper_2607_03226_b200 import workloads as wl
from test_oracle_pins import TINY, random_T, small_bands

pytestmark = pytest.mark.gpu

TOL_SWEEP = 1e-10  # max-norm relative, north_star
TOL_T_CONVERGED = 1e-8  # K, north_star


def gpu_solver(pr, **kw):
    from paper_2607_03226_b200.binding import Solver
    return Solver(pr, **kw)


def rel(a, b):
    s = np.abs(b).max()
    return np.abs(a - b).max() / s if s > 0 else np.abs(a - b).max()


def compare_state(g, r, pr, what=""):
    eg, er = g.get_e(), r.get_e()
    assert eg.shape == er.shape
    for b in range(er.shape[0]):
        assert rel(eg[b], er[b]) <= TOL_SWEEP, f"{what}: e band {b}: {rel(eg[b], er[b]):.3e}"


def compare_fields(g, r, pr, what=""):
    Tr = pr["T_ref"]
    for which in (0, 1, 2):
        a, b = g.get_T(which) - Tr, r.get_T(which) - Tr
        assert rel(a, b) <= TOL_SWEEP, f"{what}: T[{which}] {rel(a, b):.3e}"
    assert rel(g.get_q(), r.get_q()) <= TOL_SWEEP, f"{what}: q"
    if r.n_bf:
        assert rel(g.get_G(), r.get_G()) <= TOL_SWEEP, f"{what}: G"


def step_parity(pr, n_steps=3, T_init=None, mode="plain", **kw):
    r = RefSolver(pr, T_init=T_init)
    g = gpu_solver(pr, T_init=T_init, **kw)
    assert g.n_active == r.n_active and abs(g.kappa - r.kappa) <= 1e-14 * abs(r.kappa)
    for n in range(n_steps):
        r.sweep()
        g.sweep()
        compare_state(g, r, pr, f"sweep {n}")
        dr = r.update_temperature()
        dg = g.update_temperature()
        compare_fields(g, r, pr, f"update {n}")
        assert abs(dg - dr) <= 1e-9 * max(abs(dr), 1e-300) + 1e-13
        Hg, Hr = g.get_boundary_heat(), r.get_boundary_heat()
        assert np.abs(Hg - Hr).max() <= 1e-9 * max(np.abs(Hr).max(), 1e-300)
        if mode == "synthetic":
            (ir, d2r), (ig, d2g) = r.diffusion_correct(), g.diffusion_correct()
            a, b = g.get_T(0) - pr["T_ref"], r.get_T(0) - pr["T_ref"]
            assert rel(a, b) <= 1e-9, f"synthetic step {n}: {rel(a, b):.3e}"
            # the GPU CG starts from a recycled initial guess: same system, same stopping rule,
            # so it never needs noticeably more iterations than the oracle's CG from zero
            assert ig <= ir + max(2, ir // 20)
    g.close()
    r.close()


# ---- tiny meshes: every closure type, non-uniform spacing, a masked L-shape ------------------------------------------
@pytest.mark.parametrize("variant", [0, 4])  # 0: auto (single-buffered sweep), 4: double-buffered sweep
@pytest.mark.parametrize("name", [k for k in TINY if TINY[k]["kind"] == "structured"])
def test_tiny_steps(name, variant):
    pr = TINY[name]
    m = pr["mesh"]
    uniform = all(np.ptp(np.asarray(m[k], dtype=np.float64)) == 0.0 for k in ("hx", "hy", "hz"))
    if variant == 4 and not uniform:  # the double-buffered sweep is for uniform spacing: refused, not silently replaced
        from paper_2607_03226_b200.binding import NanoBTEError
        with pytest.raises(NanoBTEError) as e:
            gpu_solver(pr, sweep_variant=4)
        assert e.value.code == -11
        return
    step_parity(pr, 4, T_init=random_T(pr, 5), sweep_variant=variant)


@pytest.mark.parametrize("name", [k for k in TINY if TINY[k]["kind"] == "structured"])
def test_tiny_synthetic_steps(name):
    pr = dict(TINY[name])
    pr["bands"] = small_bands(len(pr["bands"]["C"]), 21, lo=-11.3)
    step_parity(pr, 3, T_init=random_T(pr, 6), mode="synthetic")


@pytest.mark.parametrize("name", [k for k in TINY if TINY[k]["kind"] == "structured"])
@pytest.mark.parametrize("mode", ["plain", "synthetic"])
def test_tiny_solve(name, mode):
    pr = dict(TINY[name])
    if mode == "synthetic":
        pr["bands"] = small_bands(len(pr["bands"]["C"]), 21, lo=-11.3)
    r, g = RefSolver(pr), gpu_solver(pr)
    rr, rg = r.solve(1e-11, 20000, mode), g.solve(1e-11, 20000, mode)
    assert rr["converged"] and rg["converged"]
    assert rg["iters"] == rr["iters"]
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED
    hg, hr = g.get_history()[0], r.get_history()[0]
    np.testing.assert_allclose(hg, hr, rtol=1e-6, atol=HIST_ATOL)


# ---- BASELINE.json configs[0] (full size) and configs[1] (full size), several launch shapes --------------------------------
def test_config0_gray_square_full():
    pr = wl.config_gray_square()
    step_parity(pr, 3)
    r, g = RefSolver(pr), gpu_solver(pr)
    rr, rg = r.solve(pr["tol"], pr["max_iter"]), g.solve(pr["tol"], pr["max_iter"])
    assert rr["iters"] == rg["iters"] == 35
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED
    assert np.abs(g.get_T(1) - r.get_T(1)).max() <= TOL_T_CONVERGED
    assert rel(g.get_q(), r.get_q()) <= 1e-8


@pytest.mark.parametrize("kw", [{}, {"sweep_G": 1}, {"sweep_G": 2, "sweep_threads": 64}, {"sweep_G": 4},
                                {"sweep_G": 1, "sweep_threads": 32}, {"sweep_variant": 4}, {"sweep_variant": 4, "sweep_G": 2},
                                {"sweep_variant": 4, "sweep_G": 3, "sweep_threads": 96}])
def test_config1_nongray_square_full(kw):
    pr = wl.config_nongray_square()
    step_parity(pr, 2, **kw)


def test_config1_solve():
    pr = wl.config_nongray_square(n=48)
    r, g = RefSolver(pr), gpu_solver(pr)
    rr, rg = r.solve(pr["tol"], pr["max_iter"]), g.solve(pr["tol"], pr["max_iter"])
    assert rr["converged"] and rg["converged"] and rr["iters"] == rg["iters"]
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED


# ---- cuts of configs[2] (cube) and configs[3] (finfet): several tiles and ragged tails ---------------------------------------
@pytest.mark.parametrize("n,kw", [(12, {}), (20, {"sweep_G": 1}), (20, {"sweep_G": 2}), (20, {"sweep_G": 4, "sweep_threads": 128}),
                                  (33, {"sweep_G": 2, "sweep_threads": 160}), (24, {"sweep_G": 1, "sweep_threads": 96}),
                                  (20, {"sweep_variant": 4}), (33, {"sweep_variant": 4, "sweep_G": 2, "sweep_threads": 160}),
                                  (24, {"sweep_variant": 4, "sweep_G": 3}), (17, {"sweep_variant": 3, "sweep_G": 3})])
def test_cube_cut_steps(n, kw):
    pr = wl.config_cube(n=n, B=3, n_polar=4, n_azim=8)
    step_parity(pr, 3, T_init=random_T(pr, 9), **kw)


def test_cube_cut_solve_both_modes():
    pr = wl.config_cube(n=10, B=4, n_polar=2, n_azim=8)
    Ts = {}
    for mode in ("plain", "synthetic"):
        r, g = RefSolver(pr), gpu_solver(pr)
        rr, rg = r.solve(1e-9, 3000, mode), g.solve(1e-9, 3000, mode)
        assert rr["converged"] and rg["converged"], (rr, rg)
        assert rr["iters"] == rg["iters"], (mode, rr, rg)
        assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED
        Ts[mode] = g.get_T(0)
    assert np.abs(Ts["plain"] - Ts["synthetic"]).max() < 1e-6  # P6 on the GPU side


@pytest.mark.parametrize("shape,kw", [((16, 8, 8), {}), ((32, 16, 16), {"sweep_G": 2}), ((24, 12, 12), {"sweep_G": 1}),
                                      ((32, 16, 16), {"sweep_variant": 4}), ((24, 12, 12), {"sweep_variant": 4, "sweep_G": 3})])
def test_finfet_cut_steps(shape, kw):
    nx, ny, nz = shape
    pr = wl.config_finfet(nx=nx, ny=ny, nz=nz, B=3, n_polar=2, n_azim=8)
    step_parity(pr, 3, T_init=random_T(pr, 10), mode="synthetic", **kw)


def test_finfet_cut_solve():
    pr = wl.config_finfet(nx=16, ny=8, nz=8, B=3, n_polar=2, n_azim=8)
    for mode in ("plain", "synthetic"):
        r, g = RefSolver(pr), gpu_solver(pr)
        rr, rg = r.solve(1e-9, 5000, mode), g.solve(1e-9, 5000, mode)
        assert rr["converged"] and rg["converged"], (rr, rg)
        assert rr["iters"] == rg["iters"], (mode, rr, rg)
        assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED


@pytest.mark.parametrize("which", ["cube", "finfet"])
def test_brick_closures_many_bands_and_groups(which):
    """40 bands x 16 directions per octant: five band groups of eight bands per class and more bands than lanes, i.e. the
    general loops of brick_gsum_kernel (groups beyond the four of one pass, bands beyond 32) and inflow records of every
    face type (cube: thermalizing, diffuse, specular; finfet: mixed) with 16-direction permutations."""
    pr = (wl.config_cube(n=12, B=40, n_polar=8, n_azim=16, mode="synthetic") if which == "cube"
          else wl.config_finfet(nx=16, ny=8, nz=8, B=40, n_polar=8, n_azim=16))
    step_parity(pr, 2, T_init=random_T(pr, 21), mode="synthetic")


@pytest.mark.parametrize("endseg", [None, "0", "20"])
def test_brick_long_pencils_segmentations(monkeypatch, endseg):
    """Pencils of 128 cells: the tile-dataflow sweep cuts them into 12 + 52 + 52 + 12 planes (default), evenly
    (NANOBTE_BRICK_ENDSEG=0) or with 20-plane ends; the u-face hand-over between segments and the source-plane masks of
    52-plane segments against the oracle."""
    if endseg is not None:
        monkeypatch.setenv("NANOBTE_BRICK_ENDSEG", endseg)
    pr = wl.config_finfet(nx=128, ny=16, nz=16, B=3, n_polar=2, n_azim=8)
    step_parity(pr, 2, T_init=random_T(pr, 22), mode="synthetic")


# ---- unstructured polygon meshes (BASELINE.json configs[4] family): level-scheduled sweep --------------------------------------
def test_tiny_triangles_steps():
    pr = TINY["tri4x4"]
    step_parity(pr, 4, T_init=random_T(pr, 5))


def test_tiny_triangles_synthetic_and_solve():
    pr = dict(TINY["tri4x4"])
    pr["bands"] = small_bands(2, 21, lo=-11.3)
    step_parity(pr, 3, T_init=random_T(pr, 6), mode="synthetic")
    for mode in ("plain", "synthetic"):
        r, g = RefSolver(pr), gpu_solver(pr)
        rr, rg = r.solve(1e-11, 20000, mode), g.solve(1e-11, 20000, mode)
        assert rr["converged"] and rg["converged"] and rg["iters"] == rr["iters"], (mode, rr, rg)
        assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED


@pytest.mark.parametrize("n,B,D,kw", [(24, 5, 16, {}), (40, 8, 16, {"sweep_threads": 128}), (33, 3, 8, {"sweep_G": 2}),
                                      (20, 11, 8, {"sweep_G": 4, "sweep_threads": 64})])
def test_triangles_cut_steps(n, B, D, kw):
    """Cuts of configs[4]: jittered triangles with the circular hole, several CTAs per direction, ragged band groups."""
    pr = wl.config_triangles(n=n, side=2e-6 * n / 320, B=B, D=D, hole_radius=300e-9 * n / 320)
    step_parity(pr, 3, T_init=random_T(pr, 12), **kw)


def test_triangles_cut_solve():
    pr = wl.config_triangles(n=16, side=1e-7, B=3, D=8, hole_radius=1.5e-8)
    r, g = RefSolver(pr), gpu_solver(pr)
    rr, rg = r.solve(1e-9, 4000), g.solve(1e-9, 4000)
    assert rr["converged"] and rg["converged"] and rr["iters"] == rg["iters"], (rr, rg)
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED


def test_polygon_quads_match_structured_on_gpu():
    tags = [(wl.THERMALIZING, 302.0), (wl.THERMALIZING, 299.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0)]
    bands, quad = small_bands(2, 8), wl.inplane_quadrature(8)
    ps = wl.make_structured_problem(9, 7, 1, 7e-9, 9e-9, 1.0, bands, quad, tags, [0, 1, 2, 3, 0, 0])
    pu = dict(ps)
    pu["kind"] = "unstructured"
    pu["mesh"] = wl.quads_as_unstructured(9, 7, 7e-9, 9e-9, lambda side: [0, 1, 2, 3][side], tags)
    a, b = gpu_solver(ps), gpu_solver(pu)
    for _ in range(4):
        a.sweep(); b.sweep()
        a.update_temperature(); b.update_temperature()
    assert rel(b.get_e(), a.get_e()) <= 1e-12
    assert np.abs(a.get_T(0) - b.get_T(0)).max() <= 1e-11


# ---- degenerate shapes ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(1, 1, 1), (7, 1, 1), (1, 9, 1), (5, 1, 3), (1, 1, 6), (2, 3, 1)])
def test_degenerate_shapes(shape):
    nx, ny, nz = shape
    tags = [(wl.THERMALIZING, 302.0), (wl.THERMALIZING, 297.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0)]
    quad = wl.product_quadrature(2, 4) if nz > 1 else wl.inplane_quadrature(8)
    pr = wl.make_structured_problem(nx, ny, nz, 7e-9, 9e-9, 11e-9, small_bands(2, 3), quad, tags, [0, 1, 2, 2, 3, 3],
                                    Qdot=np.full(nx * ny * nz, 3e16))
    step_parity(pr, 3)


def test_isothermal_stays_isothermal():
    pr = wl.config_cube(n=8, B=2, n_polar=2, n_azim=4, src=0.0)
    pr["mesh"]["tags"] = [(wl.THERMALIZING, 305.0), (wl.THERMALIZING, 305.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0)]
    g = gpu_solver(pr)
    res = g.solve(1e-12, 10)
    assert res["iters"] == 1 and res["last_dT"] == 0.0
    assert np.abs(g.get_e()).max() == 0.0


def test_bitwise_reproducible():
    pr = wl.config_cube(n=16, B=2, n_polar=2, n_azim=8)
    outs = []
    for _ in range(2):
        g = gpu_solver(pr)
        g.solve(1e-9, 6, "synthetic")
        outs.append((g.get_T(0).copy(), g.get_e(0, 1, 0, 4).copy()))
        g.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_set_T_and_device_getters():
    import torch
    pr = wl.config_cube(n=8, B=2, n_polar=2, n_azim=4)
    T0 = random_T(pr, 3)
    r, g = RefSolver(pr), gpu_solver(pr)
    r.set_T(T0)
    g.set_T(torch.as_tensor(T0, device="cuda"))
    r.sweep(); g.sweep()
    compare_state(g, r, pr)
    ed = g.get_e(device=True)
    assert ed.is_cuda and np.array_equal(ed.cpu().numpy(), g.get_e())
    assert rel(g.get_e(deviational=False), r.get_e(deviational=False)) <= 1e-12
    Td = g.get_T(0, device=True)
    assert np.array_equal(Td.cpu().numpy(), g.get_T(0))


def test_errors_on_gpu():
    from paper_2607_03226_b200.binding import NanoBTEError
    pr = wl.config_cube(n=6, B=2, n_polar=2, n_azim=4)
    pr["mesh"]["tags"] = [(wl.DIFFUSE, 0.0)] * 4
    g = gpu_solver(pr)
    with pytest.raises(NanoBTEError) as e:
        g.solve(1e-9, 5, "synthetic")
    assert e.value.code == -9


def test_generic_cg_kernel_matches_oracle(monkeypatch):
    """The multi-pass CG kernel (fallback for meshes whose chunk or halo does not fit the fused kernel)."""
    monkeypatch.setenv("NANOBTE_CG_GENERIC", "1")
    pr = wl.config_finfet(nx=24, ny=12, nz=12, B=3, n_polar=2, n_azim=8)
    step_parity(pr, 2, T_init=random_T(pr, 4), mode="synthetic")


def test_unstructured_fallback_kernel_matches_oracle(monkeypatch):
    """The ring + register-pipeline sweep that `create` falls back to when a mesh's level spans do not fit the staged
    kernel's rings."""
    monkeypatch.setenv("NANOBTE_UNS_PLAIN", "1")
    pr = wl.config_triangles(n=24, side=2e-6 * 24 / 320, B=5, D=16, hole_radius=300e-9 * 24 / 320)
    step_parity(pr, 3, T_init=random_T(pr, 12))


def test_general_cg_stencil_on_a_uniform_grid(monkeypatch):
    """The per-cell stencil path of the fused CG (what non-uniform and unstructured meshes use), forced on a grid that
    would take the face-uniform path."""
    monkeypatch.setenv("NANOBTE_CG_NO_UNI", "1")
    pr = wl.config_finfet(nx=24, ny=12, nz=12, B=3, n_polar=2, n_azim=8)
    step_parity(pr, 2, T_init=random_T(pr, 4), mode="synthetic")


@pytest.mark.parametrize("seed", [1, 2, 3, 4, 5, 6])
def test_random_masks(seed):
    """Random masks (holes inside pencils, isolated cells, walls of every type on interior faces) in both sweep
    variants: stresses the wall-first slot order, the padding slots and the inflow / source index packing."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = int(rng.integers(3, 12)), int(rng.integers(2, 9)), int(rng.integers(1, 7))
    active = (rng.random(nx * ny * nz) > 0.3).astype(np.uint8)
    active[int(rng.integers(0, nx * ny * nz))] = 1
    tags = [(wl.THERMALIZING, 303.0), (wl.THERMALIZING, 298.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0), (wl.MIXED, 0.0)]
    side_tags = [int(t) for t in rng.permutation(5)] + [int(rng.integers(0, 5))]
    if 0 not in side_tags and 1 not in side_tags:
        side_tags[0] = 0
    quad = wl.product_quadrature(2, 8) if nz > 1 else wl.inplane_quadrature(8)
    Q = np.where(rng.random(nx * ny * nz) > 0.6, 1e17 * rng.random(nx * ny * nz), 0.0)
    pr = wl.make_structured_problem(nx, ny, nz, 7e-9, 9e-9, 11e-9, small_bands(3, seed), quad, tags, side_tags,
                                    active=active, Qdot=Q, p_seed=seed)
    for variant in (0, 4):
        step_parity(pr, 3, T_init=random_T(pr, seed), sweep_variant=variant)


@pytest.mark.parametrize("seed", [100, 110, 121, 124, 137])
def test_random_masks_many_systems(seed):
    """Random masked boxes with 16 to 128 directions and up to 33 bands (more bands than lanes, 12 or 16 directions per
    octant, five wall types on interior faces) through the default path: the tile-dataflow sweep and its record-driven
    closure kernels, including the geometries where the mirror images of a class split and the general inflow kernel runs."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = int(rng.integers(3, 24)), int(rng.integers(2, 14)), int(rng.integers(2, 12))
    active = (rng.random(nx * ny * nz) > rng.choice([0.0, 0.1, 0.3])).astype(np.uint8)
    active[int(rng.integers(0, nx * ny * nz))] = 1
    tags = [(wl.THERMALIZING, 303.0), (wl.THERMALIZING, 298.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0), (wl.MIXED, 0.0)]
    side_tags = [int(t) for t in rng.permutation(5)] + [int(rng.integers(0, 5))]
    if 0 not in side_tags and 1 not in side_tags:
        side_tags[0] = 0
    npol, naz = [(2, 8), (4, 8), (6, 16), (8, 16)][int(rng.integers(0, 4))]
    B = int(rng.choice([3, 11, 33]))
    Q = np.where(rng.random(nx * ny * nz) > 0.6, 1e17 * rng.random(nx * ny * nz), 0.0)
    pr = wl.make_structured_problem(nx, ny, nz, 7e-9, 9e-9, 11e-9, small_bands(B, seed), wl.product_quadrature(npol, naz), tags,
                                    side_tags, active=active, Qdot=Q, p_seed=seed)
    step_parity(pr, 3, T_init=random_T(pr, seed), mode="synthetic" if seed % 2 else "plain")


def test_library_owned_memory_matches_caller_owned_workspace():
    """options.workspace == NULL: the library allocates its arena itself (cudaMalloc) -- same results, bit for bit."""
    pr = wl.config_cube(n=10, B=2, n_polar=2, n_azim=8)
    outs = []
    for own in (True, False):
        g = gpu_solver(pr, own_workspace=own)
        g.solve(1e-9, 5, "synthetic")
        outs.append((g.get_T(0).copy(), g.get_e(0, 1, 0, 3).copy()))
        g.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_finfet_mid_cut_solve_synthetic():
    """A cut large enough for the CG to run on many CTA chunks (halo recurrences, grid barrier): converged field and
    outer iteration count against the oracle."""
    pr = wl.config_finfet(nx=32, ny=16, nz=16, B=4, n_polar=2, n_azim=8)
    r, g = RefSolver(pr), gpu_solver(pr)
    rr, rg = r.solve(1e-9, 5000, "synthetic"), g.solve(1e-9, 5000, "synthetic")
    assert rr["converged"] and rg["converged"], (rr, rg)
    assert rr["iters"] == rg["iters"], (rr, rg)
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED
    hg, hr = g.get_history(), r.get_history()
    np.testing.assert_allclose(hg[0], hr[0], rtol=1e-6, atol=HIST_ATOL)
    assert (hg[1] - hr[1]).max() <= max(2, int(hr[1].max()) // 20)  # CG iterations per outer iteration: never noticeably more


def test_cg_from_zero_matches_oracle_counts(monkeypatch):
    """Without the recycled initial guess the GPU CG is the oracle's CG (from zero, unpreconditioned): the iteration
    counts agree within rounding effects, in both directions."""
    monkeypatch.setenv("NANOBTE_CG_NO_RECYCLE", "1")
    pr = wl.config_finfet(nx=24, ny=12, nz=12, B=3, n_polar=2, n_azim=8)
    r, g = RefSolver(pr), gpu_solver(pr)
    for _ in range(4):
        r.sweep(); g.sweep()
        r.update_temperature(); g.update_temperature()
        (ir, _), (ig, _) = r.diffusion_correct(), g.diffusion_correct()
        assert abs(ig - ir) <= max(2, ir // 20)
    assert rel(g.get_T(0) - pr["T_ref"], r.get_T(0) - pr["T_ref"]) <= 1e-9


# ---- fused-CG instantiations: 2, 4 and 8 cells per thread, halo batches beyond the unrolled ones ------------------------------------
@pytest.mark.parametrize("nblk,cpt", [(6, 2), (3, 4), (2, 8)])
@pytest.mark.parametrize("hook", ["", "NANOBTE_CG_NO_UNI", "NANOBTE_CG_NO_RECYCLE"])
def test_fused_cg_cells_per_thread_on_cuts(monkeypatch, nblk, cpt, hook):
    """NANOBTE_CG_NBLK caps the CTA count of the fused CG so that a cut runs the kernel instantiations the full-size
    configs use (4 cells per thread on configs 2-4; 2 and 8 on meshes around them), with the face-uniform and the
    general stencil, with and without the recycled guess: element-wise against the oracle for 3 synthetic steps."""
    monkeypatch.setenv("NANOBTE_CG_NBLK", str(nblk))
    monkeypatch.setenv("NANOBTE_CG_NO_MG", "1")
    if hook:
        monkeypatch.setenv(hook, "1")
    pr = wl.config_finfet(nx=32, ny=16, nz=16, B=3, n_polar=2, n_azim=8)
    g = gpu_solver(pr)
    assert g.info["cg_multigrid"] == 0
    assert g.info["cg_fused"] == 1 and g.info["cg_cells_per_thread"] == cpt and g.info["cg_ctas"] <= nblk, g.info
    assert g.info["cg_face_uniform"] == (0 if hook == "NANOBTE_CG_NO_UNI" else 1)
    g.close()
    step_parity(pr, 3, T_init=random_T(pr, 10), mode="synthetic")


@pytest.mark.parametrize("which,nblk", [("finfet", 0), ("finfet", 2), ("finfet", 5), ("cube20", 0), ("cube20", 4), ("cube33", 0),
                                        ("cube33", 40)])
def test_multigrid_cg_on_cuts(monkeypatch, which, nblk):
    """cg_mg_kernel (the synthetic correction's default on uniform 3-D grids) with 1, 3-4 and 7-8 level-3 aggregates per CTA
    (its slots-per-thread instantiations), on a masked grid and on lattices whose edge is not a multiple of 8 (partly
    empty aggregates, empty slots): theta after the correction element-wise against the oracle for 3 synthetic steps, and
    far fewer iterations than the oracle's unpreconditioned CG (same system, same ||r|| <= rtol ||rhs||: reading R14e')."""
    if nblk:
        monkeypatch.setenv("NANOBTE_CG_NBLK", str(nblk))
    pr = {"finfet": lambda: wl.config_finfet(nx=32, ny=16, nz=16, B=3, n_polar=2, n_azim=8),
          "cube20": lambda: wl.config_cube(n=20, B=3, n_polar=2, n_azim=8, mode="synthetic"),
          "cube33": lambda: wl.config_cube(n=33, B=2, n_polar=2, n_azim=8, mode="synthetic")}[which]()
    g, r = gpu_solver(pr), RefSolver(pr)
    assert g.info["cg_multigrid"] == 1 and g.info["cg_mg_levels"] >= 4, g.info
    T0 = random_T(pr, 21)
    g.set_T(T0); r.set_T(T0)
    for _ in range(3):
        g.sweep(); r.sweep()
        g.update_temperature(); r.update_temperature()
        (ig, _), (ir, _) = g.diffusion_correct(), r.diffusion_correct()
        assert rel(g.get_T(0) - pr["T_ref"], r.get_T(0) - pr["T_ref"]) <= 1e-9
        assert 0 < ig <= 40 and ig < ir // 3, (ig, ir)
    g.close(); r.close()


# ---- Fourier initial guess (reading R21) --------------------------------------------------------------
FOURIER_CASES = {
    "tiny": lambda name: TINY[name],
    "cube20": lambda _: wl.config_cube(n=20, B=3, n_polar=2, n_azim=8, mode="synthetic"),
    "finfet": lambda _: wl.config_finfet(nx=32, ny=16, nz=16, B=3, n_polar=2, n_azim=8),
    "square": lambda _: wl.config_nongray_square(n=24, B=3, D=8),
    "triangles": lambda _: wl.config_triangles(n=24, side=1e-7, B=3, D=8, hole_radius=1.5e-8),
}


@pytest.mark.parametrize("case", [("tiny", k) for k in TINY] + [(k, None) for k in FOURIER_CASES if k != "tiny"])
def test_fourier_guess_matches_oracle(case):
    """nanobte_init_fourier against the oracle's O9 (every CG kernel: multigrid on the 3-D uniform grids, fused elsewhere):
    the field element by element (CG to rtol 1e-12 on both sides: compared at 1e-9 like the correction), then the
    first sweep and update from it at the sweep tolerance."""
    kind, name = case
    pr = FOURIER_CASES[kind](name)
    g, r = gpu_solver(pr, T_init=random_T(pr, 31)), RefSolver(pr, T_init=random_T(pr, 31))
    if not any(t[0] == 0 for t in pr["mesh"]["tags"]):
        with pytest.raises(Exception):
            g.init_fourier()
        g.close(); r.close()
        return
    ig, ir = g.init_fourier(), r.init_fourier()
    a, b = g.get_T(0) - pr["T_ref"], r.get_T(0) - pr["T_ref"]
    assert rel(a, b) <= 1e-9, rel(a, b)
    assert 0 < ig <= ir + max(2, ir // 20)
    r.set_T(g.get_T(0))  # the same start on both sides: the sweep is compared at its own tolerance
    g.sweep(); r.sweep()
    compare_state(g, r, pr, "sweep after the Fourier guess")
    dg, dr = g.update_temperature(), r.update_temperature()
    compare_fields(g, r, pr, "update after the Fourier guess")
    assert abs(dg - dr) <= 1e-9 * abs(dr) + 1e-13
    g.close(); r.close()


def test_fourier_guess_then_solve_counts():
    """solve() from the Fourier field: the same iteration count and converged field as the oracle started the same way."""
    pr = wl.config_finfet(nx=24, ny=12, nz=12, B=4, n_polar=2, n_azim=8)
    g, r = gpu_solver(pr), RefSolver(pr)
    g.init_fourier(); r.init_fourier()
    rg, rr = g.solve(1e-9, 3000, "synthetic"), r.solve(1e-9, 3000, "synthetic")
    assert rg["converged"] and rr["converged"] and rg["iters"] == rr["iters"], (rg, rr)
    assert np.abs(g.get_T(0) - r.get_T(0)).max() <= TOL_T_CONVERGED
    g.close(); r.close()


# ---- band shards (Eq. 14) -------------------------------------------------------------------------------
@pytest.mark.parametrize("which,mode,world", [("cube", "plain", 2), ("finfet", "synthetic", 2), ("finfet", "synthetic", 3),
                                              ("triangles", "plain", 2), ("square", "plain", 4)])
def test_band_shards_on_one_gpu_match_the_unsharded_solver(which, mode, world):
    """`world` shards of the band table side by side on one GPU (they never wait for one another: the test sums their
    exported buffers where a process group would all-reduce them): after every step every shard holds the lattice
    temperature of the unsharded solver and of the oracle, the CG counts agree, and a converged run takes the same number
    of iterations."""
    from paper_2607_03226_b200.sharded import ShardedSolver
    pr = {"cube": lambda: wl.config_cube(n=12, B=5, n_polar=2, n_azim=8, mode="synthetic"),
          "finfet": lambda: wl.config_finfet(nx=24, ny=12, nz=12, B=6, n_polar=2, n_azim=8),
          "triangles": lambda: wl.config_triangles(n=16, side=1e-7, B=5, D=8, hole_radius=1.5e-8),
          "square": lambda: wl.config_nongray_square(n=24, B=6, D=8)}[which]()
    shards = [ShardedSolver(pr, r, world) for r in range(world)]
    g, r = gpu_solver(pr), RefSolver(pr)
    assert sorted(b for s in shards for b in s.bands) == list(range(len(pr["bands"]["C"])))
    for n in range(3):
        bufs = [s.local_update() for s in shards]
        tot = bufs[0].clone()
        for b in bufs[1:]:
            tot += b
        outs = [s.finish(tot, mode) for s in shards]
        g.sweep(); r.sweep()
        dg, dr = g.update_temperature(), r.update_temperature()
        ig = ir = 0
        if mode == "synthetic":
            (ig, dg), (ir, dr) = g.diffusion_correct(), r.diffusion_correct()
        Tg, Tr = g.get_T(0) - pr["T_ref"], r.get_T(0) - pr["T_ref"]
        for s, (dT, it) in zip(shards, outs):
            Ts = s.local.get_T(0) - pr["T_ref"]
            assert rel(Ts, Tg) <= 1e-9 and rel(Ts, Tr) <= 1e-9, (n, rel(Ts, Tg), rel(Ts, Tr))
            assert abs(dT - dg) <= 1e-8 * abs(dg) + 1e-13
            assert abs(it - ig) <= max(2, ig // 10)
            for which_T in (1, 2):
                assert rel(s.local.get_T(which_T) - pr["T_ref"], r.get_T(which_T) - pr["T_ref"]) <= 1e-9
            assert rel(s.local.get_q(), r.get_q()) <= 1e-9
        assert np.array_equal(shards[0].local.get_T(0), shards[-1].local.get_T(0))  # bitwise the same on every shard
    for s in shards:
        s.close()
    # converged: same count as the unsharded oracle
    shards = [ShardedSolver(pr, k, world) for k in range(world)]
    r2 = RefSolver(pr)
    rr = r2.solve(1e-9, 3000, mode)
    n, dT = 0, 1.0
    while dT >= 1e-9 and n < 3000:
        bufs = [s.local_update() for s in shards]
        tot = bufs[0].clone()
        for b in bufs[1:]:
            tot += b
        dT = max(s.finish(tot, mode)[0] for s in shards)
        n += 1
    assert rr["converged"] and n == rr["iters"], (n, rr)
    assert np.abs(shards[0].local.get_T(0) - r2.get_T(0)).max() <= TOL_T_CONVERGED
    for s in shards:
        s.close()
    g.close(); r.close(); r2.close()


def test_brick_general_inflow_kernel(monkeypatch):
    """NANOBTE_BRICK_SLOW_INFLOW=1: the closure kernel of the tile-dataflow path that looks the mirror direction up per thread
    (the fallback when the per-row records do not apply) instead of the record-based one."""
    monkeypatch.setenv("NANOBTE_BRICK_SLOW_INFLOW", "1")
    step_parity(wl.config_finfet(nx=16, ny=8, nz=8, B=3, n_polar=2, n_azim=8), 3, mode="synthetic")
    step_parity(wl.config_cube(n=12, B=3, n_polar=2, n_azim=8), 3)


def test_cg_not_converged_is_reported():
    """cg_max_iter too small: diffusion_correct and solve say NOT_CONVERGED (1) instead of OK."""
    pr = wl.config_finfet(nx=24, ny=12, nz=12, B=3, n_polar=2, n_azim=8)
    g = gpu_solver(pr, cg_max_iter=5)
    g.sweep()
    g.update_temperature()
    rc = g._lib.nanobte_diffusion_correct(g._h, None, None)
    assert rc == 1
    res = g.solve(1e-9, 3, "synthetic")
    assert not res["converged"]
    g.close()


# ---- two live structured solvers that share a kernel instantiation with different shared-memory sizes ----------------------
def test_interleaved_big_and_small_solvers():
    big = wl.config_cube(n=28, B=3, n_polar=2, n_azim=8)
    small = wl.config_cube(n=8, B=3, n_polar=2, n_azim=8)
    kw = {"sweep_G": 2, "sweep_threads": 128}
    gb, gs = gpu_solver(big, **kw), gpu_solver(small, **kw)
    rb, rs = RefSolver(big), RefSolver(small)
    assert gb.info["sweep_smem_bytes"] > 2 * gs.info["sweep_smem_bytes"]
    for _ in range(3):  # big, small, big, ...: the per-function shared-memory cap must follow the launching solver
        gb.sweep(); rb.sweep()
        gs.sweep(); rs.sweep()
        compare_state(gb, rb, big, "big")
        compare_state(gs, rs, small, "small")
        gb.update_temperature(); rb.update_temperature()
        gs.update_temperature(); rs.update_temperature()
    for s in (gb, gs, rb, rs):
        s.close()


# ---- directions exactly parallel to grid faces ---------------------------------------------------------------------------
def axis_parallel_quadrature(dim):
    if dim == 2:
        a = np.sqrt(0.5)
        s = np.array([[1, 0, 0], [a, a, 0], [0, 1, 0], [-a, a, 0], [-1, 0, 0], [-a, -a, 0], [0, -1, 0], [a, -a, 0]], dtype=np.float64)
        return {"s": s, "w": np.full(8, 2 * np.pi / 8), "dim": 2}
    a = 1.0 / np.sqrt(3.0)
    axes = [[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]]
    diag = [[sx * a, sy * a, sz * a] for sx in (1, -1) for sy in (1, -1) for sz in (1, -1)]
    s = np.array(axes + diag, dtype=np.float64)
    w = np.concatenate([np.full(6, 4 * np.pi * 0.4 / 6), np.full(8, 4 * np.pi * 0.6 / 8)])
    return {"s": s, "w": w, "dim": 3}


@pytest.mark.parametrize("shape", [(6, 5, 1), (5, 4, 3)])
@pytest.mark.parametrize("mode", ["plain", "synthetic"])
def test_axis_parallel_directions(shape, mode):
    """A component of s exactly 0 (s.n = 0 on some faces, R15): such a face carries nothing for that direction, on every
    wall type; the oracle drops the face from both sums, the CUDA path multiplies a finite cache slot by 0."""
    nx, ny, nz = shape
    tags = [(wl.THERMALIZING, 303.0), (wl.MIXED, 0.0), (wl.SPECULAR, 0.0), (wl.DIFFUSE, 0.0), (wl.SPECULAR, 0.0)]
    bands = small_bands(2, 31, lo=-11.3)
    pr = wl.make_structured_problem(nx, ny, nz, 7e-9, 7e-9, 7e-9, bands, axis_parallel_quadrature(3 if nz > 1 else 2), tags,
                                    [0, 1, 2, 3, 4, 2], Qdot=np.full(nx * ny * nz, 2e16), p_seed=5)
    step_parity(pr, 4, T_init=random_T(pr, 8), mode=mode)
