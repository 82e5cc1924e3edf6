// setup_structured.cu -- (a1) one-time setup for structured (optionally masked) grids: validation, octant
// classes, pencil/hyperplane schedule, per-cell upwind flags, boundary-closure tables, coefficient tables,
// diffusion stencil.  Everything iteration-independent is built here once.
#include <algorithm>
#include <numeric>

#include <cstdlib>

#include "brick_host.h"
#include "host_util.h"

namespace {

inline double __longlong_as_double_host(uint64_t v) { double d; std::memcpy(&d, &v, sizeof(d)); return d; }

struct Grid {
  int n[3];
  std::vector<double> hsz[3];
  std::vector<uint8_t> act;
  int dim;
  inline int cell(int i, int j, int k) const { return i + n[0] * (j + n[1] * k); }
  inline bool inside(const int c[3]) const {
    return c[0] >= 0 && c[0] < n[0] && c[1] >= 0 && c[1] < n[1] && c[2] >= 0 && c[2] < n[2];
  }
};

struct OctHost {
  int sign[3];
  std::vector<int> dirs;
  std::vector<uint2> pen;
  std::vector<int4> plane;
  std::vector<double2> tq;         // per position: .x = theta, .y = bit pattern of (info | upwind slots << 32)
  std::vector<double> qlist;       // Qdot of the source cells, position order, each hyperplane's slice padded to even
  std::vector<double> rhu;
  std::vector<double2> pen_rh;
  std::vector<int32_t> in_bf;      // inflow list: boundary face ids in consumption order
  std::vector<int32_t> bf_slot;    // [n_bf] index of the face in in_bf, or -1
  std::vector<int32_t> cell2pos;   // [n_cells]
  std::vector<int32_t> out_bf, out_pos;  // faces that are outgoing for the class and their wall cell's position, position order
  std::vector<uint8_t> out_ord;    // rank of the class among the face's outgoing classes
  int n_pen = 0, H = 0, n_pos = 0, p_max = 0, g_max = 0, q_max = 0;
};

int build(nanobte_solver *h, const nanobte_structured_mesh *m, const nanobte_bands *bands, const nanobte_quadrature *quad,
          const nanobte_tag *tags, int n_tags, const double *Qdot, const nanobte_options *opt, bool size_only,
          size_t *bytes_out) {
  if (!m || !opt) return nb_fail(h, NANOBTE_E_INVALID, "null argument");
  Grid g;
  g.n[0] = m->nx; g.n[1] = m->ny; g.n[2] = m->nz;
  if (m->nx < 1 || m->ny < 1 || m->nz < 1 || !m->hx || !m->hy || (m->nz > 1 && !m->hz)) return nb_fail(h, NANOBTE_E_INVALID, "bad grid");
  g.dim = m->nz > 1 ? 3 : 2;
  const int dim = g.dim, nside = 2 * dim;
  const int64_t nc64 = (int64_t)m->nx * m->ny * m->nz;
  if (nc64 > (int64_t)1 << 30) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "more than 2^30 cells");
  const int nc = (int)nc64;
  g.hsz[0].assign(m->hx, m->hx + m->nx);
  g.hsz[1].assign(m->hy, m->hy + m->ny);
  if (dim == 3) g.hsz[2].assign(m->hz, m->hz + m->nz); else g.hsz[2].assign(1, 1.0);  // unit depth in 2-D
  for (int a = 0; a < 3; ++a)
    for (double v : g.hsz[a])
      if (!(v > 0)) return nb_fail(h, NANOBTE_E_INVALID, "non-positive cell size");
  g.act.assign(nc, 1);
  if (m->active) for (int c = 0; c < nc; ++c) g.act[c] = m->active[c] ? 1 : 0;

  Common cm;
  int rc = nb_validate_common(h, dim, bands, quad, tags, n_tags, cm);
  if (rc) return rc;
  // band shard: the sums over the whole band table come from the caller (nanobte_options)
  if (opt->beta_total > 0.0) cm.beta = opt->beta_total;
  if (opt->Csum_total > 0.0) {
    cm.Csum = opt->Csum_total;
    if (bands->src_share == nullptr)  // source shares of the shard's bands in the whole table (R5)
      for (int b = 0; b < cm.B; ++b) cm.share[b] = cm.C[b] / cm.Csum;
  }
  if (opt->kappa_total > 0.0) cm.kappa = opt->kappa_total;
  const int B = cm.B, D = cm.D;

  GenericTables G;
  G.cell2act.assign(nc, -1);
  for (int c = 0; c < nc; ++c)
    if (g.act[c]) { G.cell2act[c] = (int)G.act2cell.size(); G.act2cell.push_back(c); }
  const int na = (int)G.act2cell.size();
  if (na == 0) return nb_fail(h, NANOBTE_E_INVALID, "no active cell");

  // ---- boundary faces ------------------------------------------------------------------------------------------
  const int nbf = m->n_bfaces;
  if (nbf < 0 || (nbf > 0 && (!m->bf_cell || !m->bf_side || !m->bf_tag))) return nb_fail(h, NANOBTE_E_INVALID, "bad boundary face arrays");
  std::vector<int32_t> facebf((size_t)nc * 6, -1);  // (cell, side) -> boundary face id
  std::vector<int> bf_axis(nbf), bf_sgn(nbf);
  G.bf_act.resize(nbf); G.bf_type.resize(nbf); G.bf_p.resize(nbf); G.bf_den.resize(nbf); G.bf_area.resize(nbf); G.bf_eps_w.resize(nbf);
  h->h_bf_tag.assign(m->bf_tag, m->bf_tag + nbf);
  for (int f = 0; f < nbf; ++f) {
    const int c = m->bf_cell[f], side = m->bf_side[f];
    if (c < 0 || c >= nc || side >= nside || !g.act[c]) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: bad cell/side", f);
    const int axis = side / 2, sgn = (side & 1) ? 1 : -1;
    int ijk[3] = {c % g.n[0], (c / g.n[0]) % g.n[1], c / (g.n[0] * g.n[1])};
    int nb[3] = {ijk[0], ijk[1], ijk[2]};
    nb[axis] += sgn;
    if (g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])]) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d is an interior face", f);
    if (facebf[(size_t)c * 6 + side] >= 0) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d listed twice", f);
    facebf[(size_t)c * 6 + side] = f;
    const int tg = m->bf_tag[f];
    if (tg < 0 || tg >= n_tags) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: bad tag", f);
    const double p = m->bf_p ? m->bf_p[f] : 0.0;
    if (p < 0 || p > 1) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: specularity outside [0,1]", f);
    bf_axis[f] = axis; bf_sgn[f] = sgn;
    G.bf_act[f] = G.cell2act[c];
    G.bf_type[f] = cm.tag_type[tg];
    G.bf_p[f] = p;
    G.bf_eps_w[f] = cm.tag_T[tg] - opt->T_ref;
    const double dx = g.hsz[0][ijk[0]], dy = g.hsz[1][ijk[1]], dz = dim == 3 ? g.hsz[2][ijk[2]] : 1.0;
    G.bf_area[f] = axis == 0 ? dy * dz : axis == 1 ? dx * dz : dx * dy;
  }
  // every exposed face of an active cell must be tagged
  for (int a = 0; a < na; ++a) {
    const int c = G.act2cell[a];
    int ijk[3] = {c % g.n[0], (c / g.n[0]) % g.n[1], c / (g.n[0] * g.n[1])};
    for (int side = 0; side < nside; ++side) {
      int nb[3] = {ijk[0], ijk[1], ijk[2]};
      nb[side / 2] += (side & 1) ? 1 : -1;
      const bool interior = g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])];
      if (!interior && facebf[(size_t)c * 6 + side] < 0)
        return nb_fail(h, NANOBTE_E_UNTAGGED, "cell %d has an exposed face (side %d) without a boundary tag", c, side);
    }
  }

  // ---- direction classes (octants / quadrants) -----------------------------------------------------------------------
  std::vector<int> dir_code(D), code2cls(8, -1);
  for (int d = 0; d < D; ++d) {
    int code = 0;
    for (int a = 0; a < dim; ++a) if (cm.s[3 * d + a] < 0) code |= 1 << a;
    dir_code[d] = code;
  }
  std::vector<OctHost> oct;
  for (int code = 0; code < 8; ++code) {
    bool used = false;
    for (int d = 0; d < D; ++d) used |= dir_code[d] == code;
    if (!used) continue;
    code2cls[code] = (int)oct.size();
    OctHost o;
    for (int a = 0; a < 3; ++a) o.sign[a] = (code >> a) & 1 ? -1 : 1;
    for (int d = 0; d < D; ++d) if (dir_code[d] == code) o.dirs.push_back(d);
    oct.push_back(std::move(o));
  }
  const int ncls = (int)oct.size();
  std::vector<int32_t> dir_cls(D);
  for (int d = 0; d < D; ++d) dir_cls[d] = code2cls[dir_code[d]];

  // ---- pencil axis: fewest holes, then longest axis ----------------------------------------------------------------------
  int pa = 0;
  {
    long best_holes = -1;
    for (int cand = 0; cand < dim; ++cand) {
      int va = cand == 0 ? 1 : 0, wa = cand == 2 ? 1 : 2;
      long holes = 0;
      for (int w = 0; w < g.n[wa]; ++w)
        for (int v = 0; v < g.n[va]; ++v) {
          int cnt = 0;
          for (int u = 0; u < g.n[cand]; ++u) {
            int c[3]; c[cand] = u; c[va] = v; c[wa] = w;
            cnt += g.act[g.cell(c[0], c[1], c[2])];
          }
          if (cnt) holes += g.n[cand] - cnt;
        }
      if (best_holes < 0 || holes < best_holes || (holes == best_holes && g.n[cand] > g.n[pa])) { best_holes = holes; pa = cand; }
    }
  }
  const int va = pa == 0 ? 1 : 0, wa = pa == 2 ? 1 : 2;
  const int nu = g.n[pa], nv = g.n[va], nw = g.n[wa];
  const bool has_w = !(dim == 2);  // in 2-D the w axis is z (one layer, no faces)
  if ((int64_t)nv * nw >= 65535) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "grid cross-section too large for the 16-bit pencil encoding");
  const int H = nu + nv + nw - 2;
  bool uniform = true;
  for (int a = 0; a < dim; ++a)
    for (double v : g.hsz[a]) uniform &= (v == g.hsz[a][0]);

  // ---- which sweep: the tile-dataflow sweep with fused moments (brick.h) on uniform 3-D grids unless the caller asks for a
  // launch shape of the hyperplane kernels (sweep_G / sweep_threads / sweep_variant 3, 4) -------------------------------------
  size_t brick_max_dirs = 0;
  for (const OctHost &o : oct) brick_max_dirs = std::max(brick_max_dirs, o.dirs.size());
  const bool brick_ok = dim == 3 && uniform && brick_max_dirs <= 16;
  if (opt->sweep_variant == 5 && !brick_ok)
    return nb_fail(h, NANOBTE_E_UNSUPPORTED, "the tile-dataflow sweep (sweep_variant 5) needs a 3-D grid with uniform spacing and at most 16 directions per octant");
  const bool use_brick = brick_ok && (opt->sweep_variant == 5 || (opt->sweep_variant == 0 && opt->sweep_G == 0 && opt->sweep_threads == 0 &&
                                                                  std::getenv("NANOBTE_NO_BRICK") == nullptr));

  // ---- pencils (physical coordinates): which exist, which touch a +-v / +-w boundary face ---------------------------------------
  std::vector<uint8_t> pen_any((size_t)nv * nw, 0), pen_wall((size_t)nv * nw, 0);
  for (int w = 0; w < nw; ++w)
    for (int v = 0; v < nv; ++v)
      for (int u = 0; u < nu; ++u) {
        int c[3]; c[pa] = u; c[va] = v; c[wa] = w;
        if (!g.act[g.cell(c[0], c[1], c[2])]) continue;
        pen_any[(size_t)v + (size_t)nv * w] = 1;
        for (int axis : {va, wa}) {
          if (axis == wa && !has_w) continue;
          for (int sgn = -1; sgn <= 1; sgn += 2) {
            int nb[3] = {c[0], c[1], c[2]};
            nb[axis] += sgn;
            if (!(g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])])) pen_wall[(size_t)v + (size_t)nv * w] = 1;
          }
        }
      }

  // ---- per class: pencils, hyperplanes, cell info, inflow lists ----------------------------------------------------------
  int n_pen_max = 0, n_pos_max = 0, p_max = 0, g_max = 0, q_max = 0;
  std::vector<uint8_t> bf_nord(nbf, 0);  // outgoing classes per face (4 in 3-D, 2 in 2-D)
  for (int ci = 0; ci < ncls; ++ci) {
    OctHost &o = oct[ci];
    auto phys = [&](int axis, int x) { return o.sign[axis] > 0 ? x : g.n[axis] - 1 - x; };
    auto cell_of = [&](int u, int v, int w) { int c[3]; c[pa] = phys(pa, u); c[va] = phys(va, v); c[wa] = phys(wa, w); return g.cell(c[0], c[1], c[2]); };
    // Slot order: wall pencils first (those with a boundary face on a +-v or +-w side somewhere along the pencil),
    // then interior pencils; each group sorted by (m = v'+w', w') with every diagonal padded to an even slot count.
    // A hyperplane's active slots are then two contiguous ranges, one per group, and its wall cells are contiguous
    // in every e row -- which is what lets the closure kernels read the walls with coalesced loads.
    std::vector<int> pen_v, pen_w, pen_of((size_t)nv * nw, -1);
    std::vector<int> first_of_m[2] = {std::vector<int>(nv + nw, 0), std::vector<int>(nv + nw, 0)};
    for (int grp = 0; grp < 2; ++grp) {
      for (int mm = 0; mm <= nv + nw - 2; ++mm) {
        if (pen_v.size() & 1) { pen_v.push_back(-1); pen_w.push_back(-1); }  // padding slot: keeps every diagonal's first slot even
        first_of_m[grp][mm] = (int)pen_v.size();
        for (int w = std::max(0, mm - nv + 1); w <= std::min(nw - 1, mm); ++w) {
          const int v = mm - w;
          const size_t pv = (size_t)phys(va, v) + (size_t)nv * phys(wa, w);
          if (!pen_any[pv] || (pen_wall[pv] ? 0 : 1) != grp) continue;
          pen_of[(size_t)v + (size_t)nv * w] = (int)pen_v.size();
          pen_v.push_back(v);
          pen_w.push_back(w);
        }
      }
      if (pen_v.size() & 1) { pen_v.push_back(-1); pen_w.push_back(-1); }
      first_of_m[grp][nv + nw - 1] = (int)pen_v.size();
    }
    o.n_pen = (int)pen_v.size();
    o.pen.resize(o.n_pen);
    o.pen_rh.resize(o.n_pen);
    for (int p = 0; p < o.n_pen; ++p) {
      const int v = pen_v[p], w = pen_w[p];
      if (v < 0) {  // padding slot: never active (its cellinfo entries stay "hole")
        o.pen[p] = make_uint2(0x3fffffffu, (uint32_t)o.n_pen | ((uint32_t)o.n_pen << 16));
        o.pen_rh[p] = make_double2(0.0, 0.0);
        continue;
      }
      int nbv = v > 0 ? pen_of[(size_t)(v - 1) + (size_t)nv * w] : -1, nbw = w > 0 ? pen_of[(size_t)v + (size_t)nv * (w - 1)] : -1;
      if (nbv < 0) nbv = o.n_pen;  // the zero slot: such a cell always carries the boundary flag of that face
      if (nbw < 0) nbw = o.n_pen;
      o.pen[p] = make_uint2((uint32_t)(v + w), (uint32_t)nbv | ((uint32_t)nbw << 16));
      o.pen_rh[p] = make_double2(1.0 / g.hsz[va][phys(va, v)], has_w ? 1.0 / g.hsz[wa][phys(wa, w)] : 0.0);
    }
    o.H = H;
    o.plane.resize(2 * (size_t)(H + 1));
    std::vector<int> wlo(H), wcnt(H), ilo(H), icnt(H), start(H);
    int base = 0;
    for (int hh = 0; hh < H; ++hh) {
      const int mlo = std::max(0, hh - nu + 1), mhi = std::min(hh, nv + nw - 2);
      wlo[hh] = first_of_m[0][mlo];
      wcnt[hh] = mhi >= mlo ? first_of_m[0][mhi + 1] - wlo[hh] : 0;
      ilo[hh] = first_of_m[1][mlo];
      icnt[hh] = mhi >= mlo ? first_of_m[1][mhi + 1] - ilo[hh] : 0;
      start[hh] = (base + 15) / 16 * 16;  // 128-byte aligned e segments, 16-byte aligned table segments (bulk TMA)
      base = start[hh] + wcnt[hh] + icnt[hh];
      o.plane[2 * hh] = make_int4(wlo[hh], wcnt[hh], ilo[hh], icnt[hh]);
      o.plane[2 * hh + 1] = make_int4(start[hh], 0, 0, 0);
      o.p_max = std::max(o.p_max, wcnt[hh] + icnt[hh]);
    }
    o.n_pos = base;
    o.tq.assign((size_t)o.n_pos + 16, make_double2(0.0, __longlong_as_double_host(8ull)));  // holes / padding
    o.cell2pos.assign(nc, -1);
    o.bf_slot.assign(nbf, -1);
    const int axes[3] = {pa, va, wa};
    for (int hh = 0; hh < H; ++hh) {
      if (o.in_bf.size() & 1) o.in_bf.push_back(-1);  // every hyperplane's inflow slice starts on an even index
      const uint32_t in_lo = (uint32_t)o.in_bf.size();
      o.plane[2 * hh + 1].y = (int)in_lo;
      if (o.qlist.size() & 1) o.qlist.push_back(0.0);
      const uint32_t q_lo = (uint32_t)o.qlist.size();
      o.plane[2 * hh + 1].z = (int)q_lo;
      for (int k = 0; k < wcnt[hh] + icnt[hh]; ++k) {  // position order: wall slots, then interior slots
        const int p = k < wcnt[hh] ? wlo[hh] + k : ilo[hh] + (k - wcnt[hh]);
        if (pen_v[p] < 0) continue;
        const int u = hh - (pen_v[p] + pen_w[p]);
        const int pos = start[hh] + k;
        const int c = cell_of(u, pen_v[p], pen_w[p]);
        if (!g.act[c]) continue;  // hole
        o.cell2pos[c] = pos;
        uint32_t flags = 0;
        const uint32_t first = (uint32_t)o.in_bf.size();
        int ijk[3] = {c % g.n[0], (c / g.n[0]) % g.n[1], c / (g.n[0] * g.n[1])};
        for (int k = 0; k < (has_w ? 3 : 2); ++k) {
          const int axis = axes[k];
          int nb[3] = {ijk[0], ijk[1], ijk[2]};
          nb[axis] -= o.sign[axis];
          const bool interior = g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])];
          if (!interior) {
            const int side = 2 * axis + (o.sign[axis] > 0 ? 0 : 1);
            const int f = facebf[(size_t)c * 6 + side];  // >= 0, checked above
            flags |= 1u << k;
            o.bf_slot[f] = (int)o.in_bf.size();
            o.in_bf.push_back(f);
          }
        }
        for (int k2 = 0; k2 < (has_w ? 3 : 2); ++k2) {  // faces this class leaves the domain through, in position order
          const int axis = axes[k2];
          int nb[3] = {ijk[0], ijk[1], ijk[2]};
          nb[axis] += o.sign[axis];
          if (!(g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])])) {
            const int f = facebf[(size_t)c * 6 + 2 * axis + (o.sign[axis] > 0 ? 1 : 0)];
            o.out_bf.push_back(f);
            o.out_pos.push_back(pos);
            o.out_ord.push_back(bf_nord[f]++);
          }
        }
        if (first - in_lo >= (1u << 13)) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "a hyperplane has more than 8191 boundary inflow faces");
        uint32_t info = flags | ((first - in_lo) << 5);
        const double qc = Qdot ? Qdot[c] : 0.0;
        if (qc != 0.0) {
          const uint32_t qi = (uint32_t)o.qlist.size() - q_lo;
          if (qi >= (1u << 14)) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "a hyperplane has more than 16383 source cells");
          info |= 16u | (qi << 18);
          o.qlist.push_back(qc);
        }
        const double th0 = opt->T_init ? opt->T_init[c] - opt->T_ref : 0.0;
        o.tq[pos] = make_double2(th0, __longlong_as_double_host((uint64_t)info | ((uint64_t)o.pen[p].y << 32)));
      }
      o.g_max = std::max(o.g_max, (int)(o.in_bf.size() - in_lo));
      o.q_max = std::max(o.q_max, (int)(o.qlist.size() - q_lo));
    }
    if (o.in_bf.size() & 1) o.in_bf.push_back(-1);
    if (o.qlist.size() & 1) o.qlist.push_back(0.0);
    o.plane[2 * (size_t)H] = make_int4(0, 0, 0, 0);
    o.plane[2 * (size_t)H + 1] = make_int4(o.n_pos, (int)o.in_bf.size(), (int)o.qlist.size(), 0);
    // reciprocal spacings along the sweep axis, in primed coordinates
    o.rhu.resize(nu);
    for (int u = 0; u < nu; ++u) o.rhu[u] = 1.0 / g.hsz[pa][phys(pa, u)];
    n_pen_max = std::max(n_pen_max, o.n_pen);
    p_max = std::max(p_max, o.p_max);
    g_max = std::max(g_max, o.g_max);
    q_max = std::max(q_max, o.q_max);
    n_pos_max = std::max(n_pos_max, o.n_pos);
  }
  const int64_t e_stride = ((int64_t)n_pos_max + 31) / 32 * 32;

  // ---- boundary closure tables -----------------------------------------------------------------------------------------------
  G.bf_sn.assign((size_t)nbf * D, 0.0);
  G.bf_mirror.assign((size_t)nbf * D, -1);
  G.bf_inidx.assign((size_t)nbf * D, -1);
  G.bf_opos.assign((size_t)nbf * D, -1);
  std::vector<int> mirror_tab((size_t)6 * D, -2);  // per side code, lazily filled
  for (int f = 0; f < nbf; ++f) {
    const int axis = bf_axis[f], sgn = bf_sgn[f], side = 2 * axis + (sgn > 0 ? 1 : 0);
    const int c = G.act2cell[G.bf_act[f]];
    double nrm[3] = {0, 0, 0};
    nrm[axis] = sgn;
    double den = 0.0;
    const bool refl = G.bf_type[f] == NANOBTE_SPECULAR || G.bf_type[f] == NANOBTE_MIXED;
    for (int d = 0; d < D; ++d) {
      const double sn = cm.s[3 * d] * nrm[0] + cm.s[3 * d + 1] * nrm[1] + cm.s[3 * d + 2] * nrm[2];
      G.bf_sn[(size_t)f * D + d] = sn;
      const OctHost &o = oct[dir_cls[d]];
      if (sn < 0) {
        den += cm.w[d] * (-sn);
        const int slot = o.bf_slot[f];
        if (slot < 0) return nb_fail(h, NANOBTE_E_INVALID, "internal: inflow face %d missing from class of direction %d", f, d);
        G.bf_inidx[(size_t)f * D + d] = slot;
        if (refl) {
          int &mj = mirror_tab[(size_t)side * D + d];
          if (mj == -2) mj = nb_find_mirror(cm, d, nrm);
          if (mj < 0) return nb_fail(h, NANOBTE_E_SPECULAR, "boundary face %d: mirror image of direction %d is not in the quadrature", f, d);
          if (std::fabs(cm.w[mj] - cm.w[d]) > 1e-13 * cm.w[d])
            return nb_fail(h, NANOBTE_E_SPECULAR, "boundary face %d: direction %d and its mirror image %d carry different weights", f, d, mj);
          G.bf_mirror[(size_t)f * D + d] = mj;
        }
      } else if (sn > 0) {
        G.bf_opos[(size_t)f * D + d] = o.cell2pos[c];
      }
    }
    G.bf_den[f] = den;
  }
  // e rows and inflow rows are class-contiguous: class c owns rows [row0[c], row0[c] + |dirs(c)|*B) in the order
  // (direction within the class, band); its inflow rows [n_in(c)] follow the same order from bin_base[c].
  G.dir_bin.resize(D); G.dir_nin.resize(D); G.dir_row0.resize(D);
  std::vector<int32_t> cls_row0(ncls);
  std::vector<int64_t> cls_bin(ncls);
  int64_t tot = 0;
  int row = 0;
  for (int ci = 0; ci < ncls; ++ci) {
    cls_row0[ci] = row;
    cls_bin[ci] = tot;
    for (int d : oct[ci].dirs) {
      G.dir_bin[d] = tot;
      G.dir_nin[d] = (int32_t)oct[ci].in_bf.size();
      G.dir_row0[d] = row;
      tot += (int64_t)B * G.dir_nin[d];
      row += B;
    }
  }
  G.bin_total = tot;
  // closure launch lists: reflecting faces (every iteration), thermalizing faces (diagnostics on demand), class directions
  std::vector<int32_t> refl_faces, therm_faces;
  for (int f = 0; f < nbf; ++f) (G.bf_type[f] == NANOBTE_THERMALIZING ? therm_faces : refl_faces).push_back(f);
  int max_cls_dirs = 0;
  for (auto &o : oct) max_cls_dirs = std::max<int>(max_cls_dirs, (int)o.dirs.size());
  std::vector<int32_t> cls_dirs((size_t)ncls * max_cls_dirs, 0);
  for (int ci = 0; ci < ncls; ++ci)
    for (size_t k = 0; k < oct[ci].dirs.size(); ++k) cls_dirs[(size_t)ci * max_cls_dirs + k] = oct[ci].dirs[k];

  // ---- per-row coefficient tables ----------------------------------------------------------------------------------------------
  std::vector<double> coef((size_t)D * B * 8, 0.0);
  G.mcoef.resize((size_t)D * B * 5);
  for (int d = 0; d < D; ++d)
    for (int b = 0; b < B; ++b) {
      const size_t sys = (size_t)G.dir_row0[d] + b;
      const double A = cm.C[b] / (cm.W * cm.tau[b]), S = cm.share[b] / cm.W, it = 1.0 / cm.tau[b];
      const double su = std::fabs(cm.s[3 * d + pa]), sv = std::fabs(cm.s[3 * d + va]), sw = has_w ? std::fabs(cm.s[3 * d + wa]) : 0.0;
      double *cf = &coef[sys * 8];
      if (uniform) {
        const double gu = cm.v[b] * su / g.hsz[pa][0], gv = cm.v[b] * sv / g.hsz[va][0], gw = has_w ? cm.v[b] * sw / g.hsz[wa][0] : 0.0;
        const double den = it + gu + gv + gw;
        cf[0] = A / den; cf[1] = S / den; cf[2] = gu / den; cf[3] = gv / den; cf[4] = gw / den;
      } else {
        cf[0] = A; cf[1] = S; cf[2] = it; cf[3] = cm.v[b] * su; cf[4] = cm.v[b] * sv; cf[5] = cm.v[b] * sw;
      }
      double *mc = &G.mcoef[sys * 5];
      mc[0] = cm.w[d] / cm.tau[b];
      mc[1] = cm.w[d];
      for (int k = 0; k < 3; ++k) mc[2 + k] = cm.v[b] * cm.w[d] * cm.s[3 * d + k];
    }

  // ---- cells: volumes, source, initial theta, diffusion stencil ------------------------------------------------------------------
  G.vol.resize(na); G.Qdot_act.resize(na); G.theta0.resize(na);
  G.cg_nf = nside;
  G.cg_xyz.assign((size_t)3 * na, 0.0);
  for (int k = 0; k < 3; ++k) G.cg_grid[k] = g.n[k];
  G.cg_nbr.assign((size_t)nside * na, 0);
  G.cg_coef.assign((size_t)nside * na, 0.0);
  G.cg_diag.assign(na, 0.0);
  G.fourier_rhs.assign(na, 0.0);
  G.cellbf_ptr.assign(na + 1, 0);
  for (int a = 0; a < na; ++a) {
    const int c = G.act2cell[a];
    int ijk[3] = {c % g.n[0], (c / g.n[0]) % g.n[1], c / (g.n[0] * g.n[1])};
    const double hh[3] = {g.hsz[0][ijk[0]], g.hsz[1][ijk[1]], dim == 3 ? g.hsz[2][ijk[2]] : 1.0};
    G.vol[a] = hh[0] * hh[1] * hh[2];
    for (int k = 0; k < 3; ++k) G.cg_xyz[3 * (size_t)a + k] = ijk[k];
    G.Qdot_act[a] = Qdot ? Qdot[c] : 0.0;
    G.fourier_rhs[a] = G.vol[a] * G.Qdot_act[a];
    G.theta0[a] = opt->T_init ? opt->T_init[c] - opt->T_ref : 0.0;
    for (int side = 0; side < nside; ++side) {
      const int axis = side / 2, sgn = (side & 1) ? 1 : -1;
      int nb[3] = {ijk[0], ijk[1], ijk[2]};
      nb[axis] += sgn;
      const double area = axis == 0 ? hh[1] * hh[2] : axis == 1 ? hh[0] * hh[2] : hh[0] * hh[1];
      G.cg_nbr[(size_t)side * na + a] = a;
      if (g.inside(nb) && g.act[g.cell(nb[0], nb[1], nb[2])]) {
        const double dist = 0.5 * (hh[axis] + g.hsz[axis][nb[axis]]);
        const double cf = cm.kappa * area / dist;
        G.cg_nbr[(size_t)side * na + a] = G.cell2act[g.cell(nb[0], nb[1], nb[2])];
        G.cg_coef[(size_t)side * na + a] = cf;
        G.cg_diag[a] += cf;
      } else {
        const int f = facebf[(size_t)c * 6 + side];
        if (G.bf_type[f] == NANOBTE_THERMALIZING) {
          G.cg_diag[a] += cm.kappa * area / (0.5 * hh[axis]);  // delta = 0 on the wall (R14e)
          G.fourier_rhs[a] += cm.kappa * area / (0.5 * hh[axis]) * G.bf_eps_w[f];  // theta = T_w - T_ref on the wall (R21)
        }
        else G.cellbf.push_back(f);
      }
    }
    G.cellbf_ptr[a + 1] = (int32_t)G.cellbf.size();
  }
  G.tagface_ptr.assign(n_tags + 1, 0);
  for (int f = 0; f < nbf; ++f) G.tagface_ptr[m->bf_tag[f] + 1]++;
  for (int t = 0; t < n_tags; ++t) G.tagface_ptr[t + 1] += G.tagface_ptr[t];
  G.tagface.resize(nbf);
  {
    std::vector<int> fill(G.tagface_ptr.begin(), G.tagface_ptr.end() - 1);
    for (int f = 0; f < nbf; ++f) G.tagface[fill[m->bf_tag[f]]++] = f;
  }

  // ---- sweep launch shape, tasks ---------------------------------------------------------------------------------------------------
  int nsys_min = 1 << 30;
  for (auto &o : oct) nsys_min = std::min<int>(nsys_min, (int)o.dirs.size() * B);
  h->uniform = uniform;
  BrickHost bh;
  if (use_brick) {
    BrickCtx bx;
    for (int a = 0; a < 3; ++a) bx.n[a] = g.n[a];
    bx.act = g.act.data(); bx.pa = pa; bx.va = va; bx.wa = wa; bx.ncls = ncls;
    for (int ci = 0; ci < ncls; ++ci) {
      for (int a = 0; a < 3; ++a) bx.sign[ci][a] = oct[ci].sign[a];
      bx.dirs.push_back(oct[ci].dirs);
    }
    bx.facebf = facebf.data(); bx.cm = &cm; bx.G = &G; bx.coef = coef.data(); bx.cls_row0 = cls_row0.data();
    bx.Qdot = Qdot; bx.T_init = opt->T_init; bx.T_ref = opt->T_ref;
    rc = nb_brick_build(h, bx, bh);
    if (rc) return rc;
    h->sweep_variant = 5; h->sweep_G = 0; h->sweep_threads = kBrickMaxS; h->sweep_rmax = 0; h->sweep_smem = nb_brick_smem_bytes();
  } else {
    rc = nb_sweep_structured_config(h, n_pen_max, p_max, g_max, q_max, H, opt->sweep_G, opt->sweep_threads, nsys_min, opt->sweep_variant, B * D);
    if (rc) return rc;
  }
  const int per_task = std::max(1, h->sweep_G);
  std::vector<int32_t> task_oct, task_row;
  for (int ci = 0; ci < ncls; ++ci) {
    h->cls_row0[ci] = cls_row0[ci];
    h->cls_nsys[ci] = (int)oct[ci].dirs.size() * B;
    h->cls_npos[ci] = oct[ci].n_pos;
    for (int r0 = 0; r0 < h->cls_nsys[ci]; r0 += per_task) {
      task_oct.push_back(ci);
      task_row.push_back(r0);
    }
  }
  h->n_tasks = use_brick ? (int)bh.tasks.size() : (int)task_oct.size();
  h->n_cls = ncls; h->bd.n_cls = ncls;
  h->n_cells = nc; h->kind = 0; h->pencil_axis = pa; h->n_planes = H;
  h->uniform = uniform;
  h->n_pos = n_pos_max; h->e_stride = e_stride;
  h->T_ref = opt->T_ref;
  h->cg_rtol = opt->cg_rtol > 0 ? opt->cg_rtol : 1e-12;
  h->cg_max_iter = opt->cg_max_iter > 0 ? opt->cg_max_iter : 100000;

  std::vector<int32_t> a2pos((size_t)ncls * na);
  for (int ci = 0; ci < ncls; ++ci)
    for (int a = 0; a < na; ++a) a2pos[(size_t)ci * na + a] = oct[ci].cell2pos[G.act2cell[a]];

  // ---- device layout: dry pass counts, real pass uploads ------------------------------------------------------------------------------
  for (int pass = 0; pass < 2; ++pass) {
    const bool dry = pass == 0;
    Arena A(h, dry);
    rc = nb_upload_generic(h, A, cm, G);
    if (rc) return nb_fail(h, rc, "device upload failed");
    std::vector<OctTab> tabs(ncls);
    for (int ci = 0; ci < ncls; ++ci) {
      OctHost &o = oct[ci];
      OctTab &t = tabs[ci];
      h->cls_outbf[ci] = A.put(o.out_bf);
      h->cls_outpos[ci] = A.put(o.out_pos);
      h->cls_outord[ci] = A.put(o.out_ord);
      h->cls_nout[ci] = (int32_t)o.out_bf.size();
      h->cls_inbf[ci] = A.put(o.in_bf);
      h->cls_nin[ci] = (int32_t)o.in_bf.size();
      h->cls_ndirs[ci] = (int32_t)o.dirs.size();
      t.pen = A.put(o.pen);
      t.plane = A.put(o.plane);
      o.qlist.resize((size_t)o.n_pos + 2 * (size_t)H + 16, 0.0);  // fixed capacity: the arena size must not depend on Qdot
      t.qlist = A.put(o.qlist);
      double2 *tq = A.put(o.tq);
      t.tq = tq;
      h->tq[ci] = tq;
      t.rhu = A.put(o.rhu);
      t.pen_rh = A.put(o.pen_rh);
      t.bin_base = cls_bin[ci];
      t.n_pen = o.n_pen; t.H = o.H; t.n_pos = o.n_pos; t.n_in = (int)o.in_bf.size();
      t.row0 = cls_row0[ci]; t.n_rows = h->cls_nsys[ci]; t.p_max = o.p_max;
    }
    h->cls_dirs = A.put(cls_dirs);
    h->max_cls_dirs = max_cls_dirs;
    h->refl_faces = A.put(refl_faces);
    h->therm_faces = A.put(therm_faces);
    h->n_refl = (int)refl_faces.size();
    h->n_therm = (int)therm_faces.size();
    h->bf_nord = A.put(bf_nord);
    h->g_partial = A.zeros<double>((size_t)4 * nbf * B);
    h->split_closures = true;
    h->d_octs = A.put(tabs);
    h->sw.task_oct = A.put(task_oct);
    h->sw.task_row = A.put(task_row);
    h->sw.coef = A.put(coef);
    h->a2pos = A.put(a2pos);
    h->dir_cls = A.put(dir_cls);
    // the tile-dataflow sweep has its own partials and (on request) eps blocks; part[] stays as the getters' scratch
    const size_t part_n = std::max<size_t>(use_brick ? 0 : (size_t)ncls * 5 * e_stride, (size_t)3 * nc + 64);
    h->part = A.zeros<double>(part_n);
    double *e = use_brick ? nullptr : A.zeros<double>((size_t)D * B * e_stride);
    if (use_brick) {
      rc = nb_brick_upload(h, A, bh);
      if (rc) return nb_fail(h, rc, "device upload failed");
    }
    h->sw.e = e; h->bd.e = e; h->bd.e_stride = e_stride;
    h->sw.bin = h->bd.bin;
    h->sw.e_stride = e_stride; h->sw.nu = nu;
    if (A.rc) return nb_fail(h, A.rc, "device upload failed");
    if (dry) {
      const size_t need = A.off + 256;
      if (size_only) { *bytes_out = need; return 0; }
      if (opt->workspace) {
        if (opt->workspace_bytes < need) return nb_fail(h, NANOBTE_E_ALLOC, "workspace of %zu B given, %zu B needed", opt->workspace_bytes, need);
        if ((uintptr_t)opt->workspace & 255) return nb_fail(h, NANOBTE_E_INVALID, "workspace must be 256-byte aligned");
        h->arena = (char *)opt->workspace; h->arena_owned = false;
      } else {
        void *p = nullptr;
        if (cudaMalloc(&p, need) != cudaSuccess) { cudaGetLastError(); return nb_fail(h, NANOBTE_E_ALLOC, "cudaMalloc of %zu B failed", need); }
        h->arena = (char *)p; h->arena_owned = true;
      }
      h->arena_bytes = need;
    }
  }
  NB_CUDA(h, cudaMallocHost((void **)&h->h_pinned, 64));
  NB_CUDA(h, cudaStreamSynchronize(h->stream));  // host vectors die here
  // initial inflow cache: thermalizing constants, zero elsewhere (eps^0 = 0, R12)
  rc = nb_launch_boundary(h, 1);
  if (rc < 0) return rc;
  NB_CUDA(h, cudaStreamSynchronize(h->stream));
  return 0;
}

}  // namespace

extern "C" int nanobte_workspace_bytes_structured(const nanobte_structured_mesh *m, const nanobte_bands *b,
                                                  const nanobte_quadrature *q, const nanobte_tag *tags, int32_t n_tags,
                                                  const nanobte_options *opt, size_t *bytes_out) {
  if (!bytes_out) return NANOBTE_E_INVALID;
  nanobte_solver tmp;
  nb_query_sm_count(&tmp);
  return build(&tmp, m, b, q, tags, n_tags, nullptr, opt, true, bytes_out);
}

extern "C" int nanobte_create_structured(const nanobte_structured_mesh *m, const nanobte_bands *b, const nanobte_quadrature *q,
                                         const nanobte_tag *tags, int32_t n_tags, const double *Qdot, const nanobte_options *opt,
                                         nanobte_solver **out) {
  if (!out) return NANOBTE_E_INVALID;
  nanobte_solver *h = new (std::nothrow) nanobte_solver();
  if (!h) return NANOBTE_E_ALLOC;
  *out = h;
  int rc = nb_check_device(h);
  if (rc) return rc;
  h->stream = opt ? (cudaStream_t)opt->stream : nullptr;
  rc = build(h, m, b, q, tags, n_tags, Qdot, opt, false, nullptr);
  if (rc < 0 && h->arena && h->arena_owned) { cudaFree(h->arena); }
  if (rc < 0) { h->arena = nullptr; }
  return rc;
}
