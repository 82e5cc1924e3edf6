"""Seeded synthetic problem generators (inputs only -- no solver arithmetic lives here).

This module is the one piece shared by the CUDA library's tests/bench and by the
CPU oracle's tests: it only *describes problems* (mesh arrays, band tables,
direction tables, boundary tags, heat source) as plain numpy arrays.  Nothing of
the method (sweep, closures, moments, CG) is computed here, and the module
imports neither the CUDA binding nor ``oracle/``.

The five named workloads are the ones in BASELINE.json ``configs`` (indices 0-4);
they stand in for the paper's own cases (PAPER.md:129-131 square with
thermalizing sides, PAPER.md:147-155 fin on a substrate with a hot spot,
PAPER.md:178/216 unstructured device meshes), whose meshes and first-principles
band tables are not available.  The recipe for each is written out in DESIGN.md
section "Input recipe".  Every generator takes size parameters so that the tests
can build small cuts of the same family.

Conventions
-----------
* structured cell id  = i + nx*(j + ny*k); side codes 0..5 = -x,+x,-y,+y,-z,+z
* direction table ``s``  is [D,3] (s_z = 0 for in-plane quadratures), ``w`` is [D]
* tag table: list of (type, T_wall); type 0 thermalizing, 1 diffuse, 2 specular,
  3 mixed (per-face specularity ``bf_p``)
"""
from __future__ import annotations

import numpy as np

HBAR = 1.054571817e-34  # J s
KB = 1.380649e-23  # J/K

THERMALIZING, DIFFUSE, SPECULAR, MIXED = 0, 1, 2, 3


# ----------------------------------------------------------------------------
# band tables
# ----------------------------------------------------------------------------
def gray_band(C=1.66e6, v=6400.0, tau=15.6e-12):
    """One band (BASELINE.json config 0: C=1.66e6 J/m^3K, v=6400 m/s, tau=15.6 ps)."""
    return {"C": np.array([C]), "v": np.array([v]), "tau": np.array([tau])}


def debye_bands(B, omega_max=8e13, T=300.0, C_total=1.66e6, v0=6400.0):
    """Debye-like table of BASELINE.json configs 1-4.

    omega_b at bin centres of [0, omega_max]; C_b ~ omega^2 * x^2 e^x/(e^x-1)^2
    (Bose-Einstein heat capacity with omega^2 DOS, x = hbar*omega/(kB*T)), scaled so
    that sum C_b = C_total; v_b = v0*(1-0.6*omega_b/omega_max);
    tau_b = 1e-9*(omega_max/omega_b)^2 clamped to [1e-12, 1e-8] s.
    """
    om = (np.arange(B) + 0.5) * omega_max / B
    x = HBAR * om / (KB * T)
    C = om**2 * x**2 * np.exp(x) / np.expm1(x) ** 2
    C = C * (C_total / C.sum())
    v = v0 * (1.0 - 0.6 * om / omega_max)
    tau = np.clip(1e-9 * (omega_max / om) ** 2, 1e-12, 1e-8)
    return {"C": C, "v": v, "tau": tau}


# ----------------------------------------------------------------------------
# angular quadratures
# ----------------------------------------------------------------------------
def inplane_quadrature(D):
    """D in-plane unit vectors, azimuth (k+1/2)*2pi/D, equal weights 2pi/D (R3/R4)."""
    phi = (np.arange(D) + 0.5) * (2.0 * np.pi / D)
    s = np.stack([np.cos(phi), np.sin(phi), np.zeros(D)], axis=1)
    w = np.full(D, 2.0 * np.pi / D)
    return {"s": s, "w": w, "dim": 2}


def product_quadrature(n_polar, n_azim, polar_axis=2):
    """Gauss-Legendre (polar cosine) x uniform half-offset azimuth (R4).

    Direction index i = j*n_azim + k, mu_j ascending; w = w_GL * 2pi/n_azim, sum w = 4pi.
    ``polar_axis`` chooses which Cartesian axis carries mu (2 = z as in the configs;
    0 is used by the slab anchor tests).
    """
    mu, wg = np.polynomial.legendre.leggauss(n_polar)
    phi = (np.arange(n_azim) + 0.5) * (2.0 * np.pi / n_azim)
    st = np.sqrt(1.0 - mu**2)
    a = (st[:, None] * np.cos(phi)[None, :]).ravel()
    b = (st[:, None] * np.sin(phi)[None, :]).ravel()
    c = np.repeat(mu, n_azim)
    if polar_axis == 2:
        s = np.stack([a, b, c], axis=1)
    elif polar_axis == 0:
        s = np.stack([c, a, b], axis=1)
    else:
        s = np.stack([b, c, a], axis=1)
    w = np.repeat(wg, n_azim) * (2.0 * np.pi / n_azim)
    return {"s": s, "w": w, "dim": 3}


# ----------------------------------------------------------------------------
# structured meshes
# ----------------------------------------------------------------------------
def structured_boundary_faces(nx, ny, nz, active=None):
    """Enumerate exposed faces (cell, side) of the active cells, in (cell, side) order."""
    dim3 = nz > 1
    act = np.ones((nz, ny, nx), dtype=bool) if active is None else \
        np.asarray(active, dtype=bool).reshape(nz, ny, nx)
    pad = np.zeros((nz + 2, ny + 2, nx + 2), dtype=bool)
    pad[1:-1, 1:-1, 1:-1] = act
    cells, sides = [], []
    ids = np.arange(nx * ny * nz).reshape(nz, ny, nx)
    shifts = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0)]
    for side, (dk, dj, di) in enumerate(shifts):
        if side >= 4 and not dim3:
            break
        nb = pad[1 + dk:1 + dk + nz, 1 + dj:1 + dj + ny, 1 + di:1 + di + nx]
        exposed = act & ~nb
        cells.append(ids[exposed])
        sides.append(np.full(exposed.sum(), side, dtype=np.uint8))
    cells = np.concatenate(cells).astype(np.int32)
    sides = np.concatenate(sides).astype(np.uint8)
    order = np.lexsort((sides, cells))
    return cells[order], sides[order]


def _structured(nx, ny, nz, hx, hy, hz, active, tag_of_face, tags, p_of_face=None):
    cells, sides = structured_boundary_faces(nx, ny, nz, active)
    bf_tag = np.asarray(tag_of_face(cells, sides), dtype=np.int32)
    bf_p = None
    if p_of_face is not None:
        bf_p = np.asarray(p_of_face(cells, sides, bf_tag), dtype=np.float64)
    return {
        "nx": nx, "ny": ny, "nz": nz,
        "hx": np.full(nx, hx) if np.isscalar(hx) else np.asarray(hx, dtype=np.float64),
        "hy": np.full(ny, hy) if np.isscalar(hy) else np.asarray(hy, dtype=np.float64),
        "hz": np.full(nz, hz) if np.isscalar(hz) else np.asarray(hz, dtype=np.float64),
        "active": None if active is None else np.ascontiguousarray(active, dtype=np.uint8).ravel(),
        "bf_cell": cells, "bf_side": sides, "bf_tag": bf_tag, "bf_p": bf_p,
        "tags": list(tags),
    }


def config_gray_square(n=20, side=200e-9, D=16, T_left=301.0, T_right=299.0,
                       wall=DIFFUSE):
    """BASELINE.json configs[0]: gray 2-D square, thermalizing left/right, diffuse top/bottom."""
    h = side / n
    tags = [(THERMALIZING, T_left), (THERMALIZING, T_right), (wall, 0.0)]

    def tag_of(cells, sides):
        return np.where(sides == 0, 0, np.where(sides == 1, 1, 2))

    mesh = _structured(n, n, 1, h, h, 1.0, None, tag_of, tags)
    return {
        "name": f"gray_square_{n}x{n}", "kind": "structured", "mesh": mesh,
        "bands": gray_band(), "quad": inplane_quadrature(D),
        "Qdot": np.zeros(n * n), "T_ref": 300.0, "mode": "plain", "tol": 1e-10, "max_iter": 2000,
    }


def config_nongray_square(n=128, side=1e-6, B=10, D=32, sigma=50e-9, peak=1e18):
    """BASELINE.json configs[1]: non-gray 2-D square, all walls thermalizing 300 K, Gaussian source."""
    h = side / n
    tags = [(THERMALIZING, 300.0)]
    mesh = _structured(n, n, 1, h, h, 1.0, None, lambda c, s: np.zeros(len(c), dtype=np.int32), tags)
    xc = (np.arange(n) + 0.5) * h
    X, Y = np.meshgrid(xc, xc, indexing="xy")  # Y is the slow (j) index
    r2 = (X - 0.5 * side) ** 2 + (Y - 0.5 * side) ** 2
    Q = peak * np.exp(-r2 / (2.0 * sigma**2))
    return {
        "name": f"nongray_square_{n}x{n}", "kind": "structured", "mesh": mesh,
        "bands": debye_bands(B), "quad": inplane_quadrature(D),
        "Qdot": Q.ravel(), "T_ref": 300.0, "mode": "plain", "tol": 1e-9, "max_iter": 2000,
    }


def config_cube(n=64, side=500e-9, B=20, n_polar=8, n_azim=16, src=1e17, mode="plain"):
    """BASELINE.json configs[2]: 3-D cube, x thermalizing 300/310 K, y diffuse, z specular,
    uniform source in the central (n/4)^3 block."""
    h = side / n
    tags = [(THERMALIZING, 300.0), (THERMALIZING, 310.0), (DIFFUSE, 0.0), (SPECULAR, 0.0)]

    def tag_of(cells, sides):
        return np.where(sides == 0, 0, np.where(sides == 1, 1, np.where(sides < 4, 2, 3)))

    mesh = _structured(n, n, n, h, h, h, None, tag_of, tags)
    lo, hi = (3 * n) // 8, (5 * n) // 8  # 24..40 for n = 64
    Q = np.zeros((n, n, n))
    Q[lo:hi, lo:hi, lo:hi] = src
    return {
        "name": f"cube_{n}^3", "kind": "structured", "mesh": mesh,
        "bands": debye_bands(B), "quad": product_quadrature(n_polar, n_azim),
        "Qdot": Q.ravel(), "T_ref": 305.0, "mode": mode, "tol": 1e-9, "max_iter": 2000,
    }


def config_finfet(nx=128, ny=64, nz=64, lx=60e-9, ly=30e-9, lz=30e-9, B=30, n_polar=6,
                  n_azim=16, src=5e18, seed=4001, mode="synthetic"):
    """BASELINE.json configs[3]: FinFET-like masked grid.

    active iff z_c < lz/3 (substrate) or |y_c - ly/2| < ly/6 (fin, full x length);
    source where fin and z_c > 5/6*lz; z = 0 faces thermalizing 300 K; every other
    boundary face mixed with p_f ~ U[0.2, 0.4] drawn from ``seed`` in face order.
    """
    hx, hy, hz = lx / nx, ly / ny, lz / nz
    zc = (np.arange(nz) + 0.5) * hz
    yc = (np.arange(ny) + 0.5) * hy
    sub = zc < lz / 3.0
    fin = np.abs(yc - 0.5 * ly) < ly / 6.0
    act = np.zeros((nz, ny, nx), dtype=bool)
    act[sub, :, :] = True
    act[:, fin, :] = True
    Q = np.zeros((nz, ny, nx))
    hot = zc > lz * 5.0 / 6.0
    Q[np.ix_(hot, fin, np.arange(nx))] = src
    Q[~act] = 0.0
    tags = [(THERMALIZING, 300.0), (MIXED, 0.0)]
    ids_k = np.arange(nx * ny * nz) // (nx * ny)

    def tag_of(cells, sides):
        return np.where((sides == 4) & (ids_k[cells] == 0), 0, 1)

    rng = np.random.default_rng(seed)

    def p_of(cells, sides, tg):
        p = rng.uniform(0.2, 0.4, size=len(cells))
        return np.where(tg == 1, p, 0.0)

    mesh = _structured(nx, ny, nz, hx, hy, hz, act, tag_of, tags, p_of)
    return {
        "name": f"finfet_{nx}x{ny}x{nz}", "kind": "structured", "mesh": mesh,
        "bands": debye_bands(B), "quad": product_quadrature(n_polar, n_azim),
        "Qdot": Q.ravel(), "T_ref": 300.0, "mode": mode, "tol": 1e-9, "max_iter": 2000,
    }


# ----------------------------------------------------------------------------
# unstructured triangles
# ----------------------------------------------------------------------------
def config_triangles(n=320, side=2e-6, B=40, D=64, hole_radius=300e-9, jitter=0.2, seed=5001):
    """BASELINE.json configs[4]: n x n quads -> 2 triangles each (diagonal by coin flip),
    interior nodes jittered by U[-jitter, jitter]*h per coordinate, triangles whose
    centroid lies within ``hole_radius`` of the centre dropped.  x = 0 thermalizing
    300 K, x = L thermalizing 305 K, y walls specular, hole diffuse."""
    rng = np.random.default_rng(seed)
    h = side / n
    ix, iy = np.meshgrid(np.arange(n + 1), np.arange(n + 1), indexing="xy")
    gx, gy = ix * h, iy * h
    gx[ix == n] = side
    gy[iy == n] = side
    xy = np.stack([gx.ravel(), gy.ravel()], axis=1)
    interior = ((ix > 0) & (ix < n) & (iy > 0) & (iy < n)).ravel()
    jit = rng.uniform(-jitter, jitter, size=xy.shape) * h
    xy = xy + jit * interior[:, None]
    flip = rng.integers(0, 2, size=(n, n)).astype(bool)
    ii, jj = np.meshgrid(np.arange(n), np.arange(n), indexing="xy")
    n00 = (ii + (n + 1) * jj).ravel()
    n10, n01, n11 = n00 + 1, n00 + (n + 1), n00 + (n + 2)
    f = flip.ravel()
    # diagonal n00-n11 (f False) or n10-n01 (f True); all triangles counter-clockwise
    t1 = np.where(f[:, None], np.stack([n00, n10, n01], 1), np.stack([n00, n10, n11], 1))
    t2 = np.where(f[:, None], np.stack([n10, n11, n01], 1), np.stack([n00, n11, n01], 1))
    tri = np.empty((2 * n * n, 3), dtype=np.int64)
    tri[0::2], tri[1::2] = t1, t2
    cen = xy[tri].mean(axis=1)
    keep = np.hypot(cen[:, 0] - 0.5 * side, cen[:, 1] - 0.5 * side) >= hole_radius
    tri = tri[keep]
    cen = cen[keep]
    # boundary edges = edges used by exactly one triangle
    e = np.concatenate([tri[:, [0, 1]], tri[:, [1, 2]], tri[:, [2, 0]]])
    key = np.sort(e, axis=1)
    kk = key[:, 0] * (n + 1) ** 2 + key[:, 1]
    uniq, inv, cnt = np.unique(kk, return_inverse=True, return_counts=True)
    bmask = cnt[inv] == 1
    bf_nodes = e[bmask]
    mid = xy[bf_nodes].mean(axis=1)
    eps = 1e-6 * h
    tag = np.full(len(bf_nodes), 3, dtype=np.int32)  # hole
    tag[np.abs(mid[:, 1]) < eps] = 2
    tag[np.abs(mid[:, 1] - side) < eps] = 2
    tag[np.abs(mid[:, 0]) < eps] = 0
    tag[np.abs(mid[:, 0] - side) < eps] = 1
    tags = [(THERMALIZING, 300.0), (THERMALIZING, 305.0), (SPECULAR, 0.0), (DIFFUSE, 0.0)]
    ncell = len(tri)
    mesh = {
        "dim": 2, "n_nodes": len(xy), "n_cells": ncell,
        "xy": np.ascontiguousarray(xy, dtype=np.float64),
        "cell_ptr": (3 * np.arange(ncell + 1)).astype(np.int32),
        "cell_nodes": np.ascontiguousarray(tri.ravel(), dtype=np.int32),
        "bf_nodes": np.ascontiguousarray(bf_nodes, dtype=np.int32),
        "bf_tag": tag, "bf_p": None, "tags": tags,
    }
    return {
        "name": f"triangles_{n}x{n}", "kind": "unstructured", "mesh": mesh,
        "bands": debye_bands(B), "quad": inplane_quadrature(D),
        "Qdot": np.zeros(ncell), "T_ref": 302.5, "mode": "plain", "tol": 1e-9, "max_iter": 2000,
    }


def quads_as_unstructured(nx, ny, hx, hy, tag_of_side, tags):
    """A plain nx x ny quad grid written in the unstructured (polygon CSR) form; used to
    cross-check the unstructured code paths against the structured ones on identical cells."""
    gx, gy = np.meshgrid(np.arange(nx + 1) * hx, np.arange(ny + 1) * hy, indexing="xy")
    xy = np.stack([gx.ravel(), gy.ravel()], axis=1)
    ii, jj = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    n00 = (ii + (nx + 1) * jj).ravel()
    quads = np.stack([n00, n00 + 1, n00 + nx + 2, n00 + nx + 1], axis=1)
    bf, tg = [], []
    for i in range(nx):
        bf.append((i + 1, i)); tg.append(tag_of_side(2))  # bottom, y = 0
        top = (nx + 1) * ny
        bf.append((top + i, top + i + 1)); tg.append(tag_of_side(3))
    for j in range(ny):
        bf.append(((nx + 1) * j, (nx + 1) * (j + 1))); tg.append(tag_of_side(0))
        bf.append(((nx + 1) * (j + 1) + nx, (nx + 1) * j + nx)); tg.append(tag_of_side(1))
    return {
        "dim": 2, "n_nodes": len(xy), "n_cells": nx * ny, "xy": xy,
        "cell_ptr": (4 * np.arange(nx * ny + 1)).astype(np.int32),
        "cell_nodes": np.ascontiguousarray(quads.ravel(), dtype=np.int32),
        "bf_nodes": np.asarray(bf, dtype=np.int32), "bf_tag": np.asarray(tg, dtype=np.int32),
        "bf_p": None, "tags": list(tags),
    }


# ----------------------------------------------------------------------------
# registry: BASELINE.json configs[0..4]
# ----------------------------------------------------------------------------
CONFIGS = {
    "gray_square": config_gray_square,          # configs[0]
    "nongray_square": config_nongray_square,    # configs[1]
    "cube": config_cube,                        # configs[2]
    "finfet": config_finfet,                    # configs[3]
    "triangles": config_triangles,              # configs[4]
}


def n_active(problem):
    m = problem["mesh"]
    if problem["kind"] == "unstructured":
        return int(m["n_cells"])
    if m["active"] is None:
        return int(m["nx"] * m["ny"] * m["nz"])
    return int(np.count_nonzero(m["active"]))


def n_updates(problem):
    """cell x band x direction updates in one sweep (the unit of BASELINE.json's metric)."""
    return n_active(problem) * len(problem["bands"]["C"]) * len(problem["quad"]["w"])


# ----------------------------------------------------------------------------
# small generic builders used by the tests
# ----------------------------------------------------------------------------
def make_structured_problem(nx, ny, nz, hx, hy, hz, bands, quad, tags, side_tags, active=None,
                            Qdot=None, T_ref=300.0, p_seed=None, p_range=(0.2, 0.8), name="custom"):
    """Structured problem with one tag id per side code (``side_tags[side]``); faces exposed by
    the mask take ``side_tags[side]`` of the side they face.  Mixed faces draw p from ``p_seed``."""
    rng = np.random.default_rng(p_seed) if p_seed is not None else None
    st = np.asarray(side_tags)

    def tag_of(cells, sides):
        return st[sides]

    def p_of(cells, sides, tg):
        types = np.array([tags[t][0] for t in tg])
        p = rng.uniform(p_range[0], p_range[1], size=len(cells)) if rng is not None else np.full(len(cells), 0.5)
        return np.where(types == MIXED, p, 0.0)

    need_p = any(t[0] == MIXED for t in tags)
    mesh = _structured(nx, ny, nz, hx, hy, hz, active, tag_of, tags, p_of if need_p else None)
    n = nx * ny * nz
    return {
        "name": name, "kind": "structured", "mesh": mesh, "bands": bands, "quad": quad,
        "Qdot": np.zeros(n) if Qdot is None else np.asarray(Qdot, dtype=np.float64).ravel(),
        "T_ref": T_ref, "mode": "plain", "tol": 1e-10, "max_iter": 5000,
    }
