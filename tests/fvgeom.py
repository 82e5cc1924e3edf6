"""Test-side finite-volume geometry + dense assembly (numpy, tiny meshes only).

Written independently of oracle/ and of the CUDA library: it derives, from the raw mesh
arrays of a workloads "problem" dict, the list of faces (owner, neighbour, area, outward
normal, distances) and from those the dense matrices that *define* what the method solves:

  * K_i      unit advection operator of direction i
  * A_{b,i}  = I/tau_b + v_b K_i                              (Eq. 13)
  * the global fixed-point system in (eps, theta)             (Eq. 4-6)
  * the two-point-flux diffusion matrix of the synthetic step (Eq. 10)

Used by the oracle pins P1, P2, P5, P6 (dense brute force) -- a different route to the
numbers than the oracle's upwind-ordered substitution.
"""
from __future__ import annotations

import numpy as np


class Geom:
    """faces: arrays over (cell, local face): owner a, nbr (active idx or -1), bf (index or -1),
    area, normal[3], dist (centroid-centroid, or centroid-face for boundary faces)."""

    def __init__(self, problem):
        m = problem["mesh"]
        self.problem = problem
        if problem["kind"] == "structured":
            self._structured(m)
        else:
            self._polygons(m)
        self.tags = m["tags"]
        self.bf_tag = np.asarray(m["bf_tag"])
        self.bf_p = np.zeros(len(self.bf_tag)) if m["bf_p"] is None else np.asarray(m["bf_p"], dtype=float)
        self.bf_type = np.array([self.tags[t][0] for t in self.bf_tag])
        self.bf_Tw = np.array([self.tags[t][1] for t in self.bf_tag])
        # map boundary face -> (owner, normal, area)
        nb = len(self.bf_tag)
        self.bf_owner = np.full(nb, -1)
        self.bf_normal = np.zeros((nb, 3))
        self.bf_area = np.zeros(nb)
        for (a, nbr, bf, A, n, d) in self.faces:
            if bf >= 0:
                self.bf_owner[bf] = a
                self.bf_normal[bf] = n
                self.bf_area[bf] = A
        assert (self.bf_owner >= 0).all()

    # -- structured ---------------------------------------------------------------------------
    def _structured(self, m):
        nx, ny, nz = m["nx"], m["ny"], m["nz"]
        self.dim = 3 if nz > 1 else 2
        act = np.ones(nx * ny * nz, bool) if m["active"] is None else np.asarray(m["active"], bool)
        self.act2cell = np.flatnonzero(act)
        self.cell2act = -np.ones(nx * ny * nz, int)
        self.cell2act[self.act2cell] = np.arange(len(self.act2cell))
        self.n_cells = nx * ny * nz
        self.n_act = len(self.act2cell)
        bfmap = {(int(c), int(s)): k for k, (c, s) in enumerate(zip(m["bf_cell"], m["bf_side"]))}
        self.vol = np.zeros(self.n_act)
        self.faces = []
        hs = [m["hx"], m["hy"], m["hz"]]
        for a, c in enumerate(self.act2cell):
            idx = [c % nx, (c // nx) % ny, c // (nx * ny)]
            h = [hs[0][idx[0]], hs[1][idx[1]], hs[2][idx[2]] if self.dim == 3 else 1.0]
            self.vol[a] = h[0] * h[1] * h[2]
            for side in range(2 * self.dim):
                ax, sg = side // 2, (1 if side % 2 else -1)
                n = np.zeros(3)
                n[ax] = sg
                A = self.vol[a] / h[ax]
                j = list(idx)
                j[ax] += sg
                nbr = -1
                dist = 0.5 * h[ax]
                if 0 <= j[0] < nx and 0 <= j[1] < ny and 0 <= j[2] < nz:
                    cn = j[0] + nx * (j[1] + ny * j[2])
                    if act[cn]:
                        nbr = self.cell2act[cn]
                        dist = 0.5 * (h[ax] + hs[ax][j[ax]])
                bf = bfmap.get((int(c), side), -1) if nbr < 0 else -1
                self.faces.append((a, nbr, bf, A, n, dist))

    # -- polygons -----------------------------------------------------------------------------
    def _polygons(self, m):
        self.dim = 2
        xy = np.asarray(m["xy"], float)
        ptr, nodes = m["cell_ptr"], m["cell_nodes"]
        nc = m["n_cells"]
        self.n_cells = self.n_act = nc
        self.act2cell = np.arange(nc)
        self.cell2act = np.arange(nc)
        bfmap = {tuple(sorted((int(a), int(b)))): k for k, (a, b) in enumerate(m["bf_nodes"])}
        edge_owner = {}
        cen = np.zeros((nc, 2))
        self.vol = np.zeros(nc)
        polys = []
        for c in range(nc):
            P = xy[nodes[ptr[c]:ptr[c + 1]]]
            x, y = P[:, 0], P[:, 1]
            xn, yn = np.roll(x, -1), np.roll(y, -1)
            cr = x * yn - xn * y
            A = 0.5 * cr.sum()
            self.vol[c] = A
            cen[c] = [((x + xn) * cr).sum() / (6 * A), ((y + yn) * cr).sum() / (6 * A)]
            polys.append(nodes[ptr[c]:ptr[c + 1]])
            for k in range(len(P)):
                key = tuple(sorted((int(polys[c][k]), int(polys[c][(k + 1) % len(P)]))))
                edge_owner.setdefault(key, []).append(c)
        self.centroid = cen
        self.faces = []
        for c in range(nc):
            pn = polys[c]
            for k in range(len(pn)):
                n0, n1 = int(pn[k]), int(pn[(k + 1) % len(pn)])
                e = xy[n1] - xy[n0]
                L = np.hypot(*e)
                n = np.array([e[1] / L, -e[0] / L, 0.0])
                key = tuple(sorted((n0, n1)))
                owners = edge_owner[key]
                if len(owners) == 2:
                    nbr = owners[0] if owners[1] == c else owners[1]
                    dist = np.hypot(*(cen[nbr] - cen[c]))
                    bf = -1
                else:
                    nbr = -1
                    dist = float((xy[n0] - cen[c]) @ n[:2])
                    bf = bfmap.get(key, -1)
                self.faces.append((c, nbr, bf, L, n, dist))

    # -- dense operators ----------------------------------------------------------------------
    def K(self, s_i):
        """Unit advection operator of direction s_i (first-order upwind) on interior faces, plus the
        list of boundary inflow terms [(a, bf, |g|)] that go to the right-hand side."""
        K = np.zeros((self.n_act, self.n_act))
        binflow = []
        for (a, nbr, bf, A, n, d) in self.faces:
            g = A * float(np.dot(s_i, n)) / self.vol[a]
            if g > 0:
                K[a, a] += g
            elif g < 0:
                if nbr >= 0:
                    K[a, nbr] += g
                else:
                    binflow.append((a, bf, -g))
        return K, binflow

    def boundary_values(self, eps_prev, T_ref):
        """O3 boundary values [n_bf, B, D] from the previous iterate eps_prev [B, D, n_act]
        (thermalizing / diffuse / specular / mixed), plus the diffuse averages G [n_bf, B]."""
        pr = self.problem
        Cb = np.asarray(pr["bands"]["C"])
        s, w = np.asarray(pr["quad"]["s"]), np.asarray(pr["quad"]["w"])
        W = w.sum()
        B, D = len(Cb), len(w)
        nb = len(self.bf_tag)
        out = np.zeros((nb, B, D))
        G = np.zeros((nb, B))
        for f in range(nb):
            a, n, typ, p = self.bf_owner[f], self.bf_normal[f], self.bf_type[f], self.bf_p[f]
            sn = s @ n
            inc, outg = sn < 0, sn > 0
            den = (w[inc] * -sn[inc]).sum()
            G[f] = (eps_prev[:, outg, a] * (w[outg] * sn[outg])[None, :]).sum(axis=1) / den
            for i in np.flatnonzero(inc):
                if typ == 0:
                    out[f, :, i] = Cb * (self.bf_Tw[f] - T_ref) / W
                elif typ == 1:
                    out[f, :, i] = G[f]
                else:
                    r = s[i] - 2 * sn[i] * n
                    j = int(np.argmin(((s - r) ** 2).sum(axis=1)))
                    assert ((s[j] - r) ** 2).sum() < 1e-18
                    spec = eps_prev[:, j, a]
                    out[f, :, i] = spec if typ == 2 else p * spec + (1 - p) * G[f]
        return out, G

    def dense_sweep(self, theta, eps_prev):
        """eps^{n+1} [B, D, n_act] by dense LAPACK solves of (I/tau_b + v_b K_i) eps = rhs."""
        pr = self.problem
        Cb, vb, tb = (np.asarray(pr["bands"][k]) for k in ("C", "v", "tau"))
        s, w = np.asarray(pr["quad"]["s"]), np.asarray(pr["quad"]["w"])
        W = w.sum()
        B, D = len(Cb), len(w)
        Q = np.asarray(pr["Qdot"])[self.act2cell]
        bcv, _ = self.boundary_values(eps_prev, pr["T_ref"])
        out = np.zeros((B, D, self.n_act))
        for i in range(D):
            K, binflow = self.K(s[i])
            for b in range(B):
                A = np.eye(self.n_act) / tb[b] + vb[b] * K
                rhs = Cb[b] * theta / (W * tb[b]) + Q * Cb[b] / (W * Cb.sum())
                for (a, bf, g) in binflow:
                    rhs[a] += vb[b] * g * bcv[bf, b, i]
                out[b, i] = np.linalg.solve(A, rhs)
        return out

    def moments(self, eps):
        pr = self.problem
        Cb, vb, tb = (np.asarray(pr["bands"][k]) for k in ("C", "v", "tau"))
        s, w = np.asarray(pr["quad"]["s"]), np.asarray(pr["quad"]["w"])
        E = np.einsum("i,bic->bc", w, eps)
        theta_SI = (E / tb[:, None]).sum(0) / (Cb / tb).sum()
        theta_en = E.sum(0) / Cb.sum()
        q = np.einsum("b,i,ik,bic->ck", vb, w, s, eps)
        return theta_SI, theta_en, q

    def cell_balance_residual(self, eps, bcv, theta_SI, theta_old):
        """P5: per-cell  sum_f A F_f + V beta (theta_SI - theta_old) - V Qdot, and the scale
        sum_f |A F_f| it should be compared with."""
        pr = self.problem
        Cb, vb, tb = (np.asarray(pr["bands"][k]) for k in ("C", "v", "tau"))
        s, w = np.asarray(pr["quad"]["s"]), np.asarray(pr["quad"]["w"])
        Q = np.asarray(pr["Qdot"])[self.act2cell]
        beta = (Cb / tb).sum()
        net = np.zeros(self.n_act)
        scale = np.zeros(self.n_act)
        for (a, nbr, bf, A, n, d) in self.faces:
            sn = s @ n
            if nbr >= 0:
                ef = np.where(sn[None, :] > 0, eps[:, :, a], eps[:, :, nbr])
            else:
                ef = np.where(sn[None, :] > 0, eps[:, :, a], bcv[bf])
            F = np.einsum("b,i,bi->", vb, w * sn, ef)
            net[a] += A * F
            scale[a] += abs(A * F)
        res = net + self.vol * beta * (theta_SI - theta_old) - self.vol * Q
        return res, scale

    def reflecting_leak(self, eps, bcv):
        """Per cell: sum over its diffuse / specular / mixed boundary faces of A_f F_f, the net heat
        that left through a wall that should carry none (non-zero only because the wall values lag,
        DESIGN.md reading R14c')."""
        pr = self.problem
        vb = np.asarray(pr["bands"]["v"])
        s, w = np.asarray(pr["quad"]["s"]), np.asarray(pr["quad"]["w"])
        leak = np.zeros(self.n_act)
        for (a, nbr, bf, A, n, d) in self.faces:
            if nbr >= 0 or self.bf_type[bf] == 0:
                continue
            sn = s @ n
            ef = np.where(sn[None, :] > 0, eps[:, :, a], bcv[bf])
            leak[a] += A * np.einsum("b,i,bi->", vb, w * sn, ef)
        return leak

    def diffusion_matrix(self, kappa):
        M = np.zeros((self.n_act, self.n_act))
        for (a, nbr, bf, A, n, d) in self.faces:
            if nbr >= 0:
                M[a, a] += kappa * A / d
                M[a, nbr] -= kappa * A / d
            elif self.bf_type[bf] == 0:
                M[a, a] += kappa * A / d
        return M

    def to_active(self, field):
        return np.asarray(field)[..., self.act2cell]

    # -- global fixed point (P2) ----------------------------------------------------------------
    def fixed_point(self):
        """Solve, in one sparse direct solve, the coupled linear system the source iteration
        converges to: unknowns x = [eps_{b,i,a} ... , theta_a ...] with

          (1/tau_b + v_b sum_out g) eps_bia - v_b sum_in |g| eps^up - C_b theta_a/(W tau_b) = S_ba
          beta theta_a - sum_b (1/tau_b) sum_i w_i eps_bia = 0                       (Eq. 5 with Eq. 6 at n -> inf)

        and eps^up = neighbour value, or the O3 boundary closure written with eps^n = eps^{n+1}.
        Returns (eps [B, D, n_act], theta [n_act])."""
        import scipy.sparse as sp
        import scipy.sparse.linalg as spla

        pr = self.problem
        Cb, vb, tb = (np.asarray(pr["bands"][k], float) for k in ("C", "v", "tau"))
        s, w = np.asarray(pr["quad"]["s"], float), np.asarray(pr["quad"]["w"], float)
        W = w.sum()
        B, D, na = len(Cb), len(w), self.n_act
        Q = np.asarray(pr["Qdot"], float)[self.act2cell]
        beta = (Cb / tb).sum()
        T_ref = pr["T_ref"]
        ne = B * D * na

        def idx(b, i, a):
            return (b * D + i) * na + a

        rows, cols, vals = [], [], []
        rhs = np.zeros(ne + na)

        def add(r, c, v):
            rows.append(r); cols.append(c); vals.append(v)

        for b in range(B):
            for i in range(D):
                for a in range(na):
                    r = idx(b, i, a)
                    add(r, r, 1.0 / tb[b])
                    add(r, ne + a, -Cb[b] / (W * tb[b]))
                    rhs[r] += Q[a] * Cb[b] / (W * Cb.sum())
        for (a, nbr, bf, A, n, d) in self.faces:
            sn = s @ n
            g = A * sn / self.vol[a]
            if nbr < 0:
                typ, p = self.bf_type[bf], self.bf_p[bf]
                inc, outg = sn < 0, sn > 0
                den = (w[inc] * -sn[inc]).sum()
            for i in range(D):
                for b in range(B):
                    r = idx(b, i, a)
                    if g[i] > 0:
                        add(r, r, vb[b] * g[i])
                    elif g[i] < 0:
                        c = -vb[b] * (-g[i])
                        if nbr >= 0:
                            add(r, idx(b, i, nbr), c)
                        elif typ == 0:
                            rhs[r] -= c * Cb[b] * (self.bf_Tw[bf] - T_ref) / W
                        else:
                            fs = 1.0 if typ == 2 else (0.0 if typ == 1 else p)
                            if fs != 0.0:
                                rv = s[i] - 2 * sn[i] * n
                                j = int(np.argmin(((s - rv) ** 2).sum(axis=1)))
                                add(r, idx(b, j, a), c * fs)
                            if fs != 1.0:
                                for j in np.flatnonzero(outg):
                                    add(r, idx(b, j, a), c * (1 - fs) * w[j] * sn[j] / den)
        for a in range(na):
            add(ne + a, ne + a, beta)
            for b in range(B):
                for i in range(D):
                    add(ne + a, idx(b, i, a), -w[i] / tb[b])
        M = sp.csc_matrix((vals, (rows, cols)), shape=(ne + na, ne + na))
        x = spla.spsolve(M, rhs)
        return x[:ne].reshape(B, D, na), x[ne:]
