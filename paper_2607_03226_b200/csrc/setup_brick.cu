// setup_brick.cu -- (a1) one-time setup of the tile-dataflow sweep (brick.h): tiles that follow the mask, segments,
// tasks in topological order with their up/downstream links, per-class cell tables and flags, the inflow / wall row
// spaces, the closure tables in those row spaces, and the per-(class, group) coefficient blocks.
#include <algorithm>
#include <cstdlib>
#include <numeric>

#include "brick_host.h"

namespace {

// Cuts of one cross-section axis: at every change of the axis' activity signature (so that walls of box-shaped masks
// fall on tile edges and the tiles have no walls inside), then every interval longer than 8 in near-equal pieces.
// A mask whose signature changes almost everywhere would shred the axis: then plain 8-wide tiles (walls inside the
// tiles go through the IRR stream).
std::vector<int> axis_cuts(int n, const std::vector<std::vector<uint8_t>> &sig) {
  std::vector<int> marks{0};
  for (int x = 1; x < n; ++x)
    if (sig[x] != sig[x - 1]) marks.push_back(x);
  marks.push_back(n);
  if ((int)marks.size() - 1 > 2 * ((n + kBrickTile - 1) / kBrickTile) + 2) marks = {0, n};
  std::vector<int> cuts{0};
  for (size_t k = 0; k + 1 < marks.size(); ++k) {
    const int len = marks[k + 1] - marks[k], pieces = (len + kBrickTile - 1) / kBrickTile;
    for (int p = 1; p <= pieces; ++p) cuts.push_back(marks[k] + (int)((int64_t)len * p / pieces));
  }
  return cuts;
}

}  // namespace

int nb_brick_build(nanobte_solver *h, const BrickCtx &x, BrickHost &bh) {
  const int nu = x.n[x.pa], nv = x.n[x.va], nw = x.n[x.wa];
  const int B = x.cm->B, D = x.cm->D, ncls = x.ncls, nbf = (int)x.G->bf_act.size(), na = (int)x.G->act2cell.size();
  auto cell_phys = [&](int u, int v, int w) { int c[3]; c[x.pa] = u; c[x.va] = v; c[x.wa] = w; return c[0] + x.n[0] * (c[1] + x.n[1] * c[2]); };
  auto active = [&](int u, int v, int w) { return u >= 0 && u < nu && v >= 0 && v < nv && w >= 0 && w < nw && x.act[cell_phys(u, v, w)]; };

  // ---- tiles and segments (physical coordinates; the same lattice for every class) --------------------------------------------
  std::vector<std::vector<uint8_t>> sigv(nv, std::vector<uint8_t>(nw, 0)), sigw(nw, std::vector<uint8_t>(nv, 0));
  for (int w = 0; w < nw; ++w)
    for (int v = 0; v < nv; ++v) {
      uint8_t any = 0;
      for (int u = 0; u < nu && !any; ++u) any = x.act[cell_phys(u, v, w)];
      sigv[v][w] = any;
      sigw[w][v] = any;
    }
  const std::vector<int> vcut = axis_cuts(nv, sigv), wcut = axis_cuts(nw, sigw);
  const int NTv = (int)vcut.size() - 1, NTw = (int)wcut.size() - 1;
  int nseg = std::max(1, (nu + 16) / 32);
  std::vector<int> ucut(nseg + 1);
  for (int k = 0; k <= nseg; ++k) ucut[k] = (int)((int64_t)nu * k / nseg);
  // Long pencils: a short segment at either end (the last tasks of a sweep are then short ones, and the ragged end of the
  // launch, when fewer tasks are left than CTAs, is half as long: config 4 1.473 -> 1.448 ms), the rest in segments of at
  // most 52 planes (a task's source-plane mask has 64 bits).  NANOBTE_BRICK_ENDSEG=n sets the end length, 0 = even segments.
  {
    int e = 12;
    if (const char *env = std::getenv("NANOBTE_BRICK_ENDSEG")) e = std::atoi(env);
    if (e > 0 && e <= 32 && nu >= 112) {
      const int mid = nu - 2 * e, nm = (mid + 51) / 52;
      nseg = nm + 2;
      ucut.assign(nseg + 1, 0);
      ucut[1] = e;
      for (int k = 1; k <= nm; ++k) ucut[1 + k] = e + (int)((int64_t)mid * k / nm);
      ucut[nseg] = nu;
    }
  }
  // which (tile, segment) boxes hold an active cell
  std::vector<uint8_t> box_on((size_t)NTv * NTw * nseg, 0);
  auto box = [&](int J, int K, int sg) { return ((size_t)sg * NTw + K) * NTv + J; };
  for (int sg = 0; sg < nseg; ++sg)
    for (int K = 0; K < NTw; ++K)
      for (int J = 0; J < NTv; ++J) {
        uint8_t any = 0;
        for (int u = ucut[sg]; u < ucut[sg + 1] && !any; ++u)
          for (int w = wcut[K]; w < wcut[K + 1] && !any; ++w)
            for (int v = vcut[J]; v < vcut[J + 1] && !any; ++v) any = x.act[cell_phys(u, v, w)];
        box_on[box(J, K, sg)] = any;
      }

  // ---- band groups per class ------------------------------------------------------------------------------------------------------
  bh.ncls = ncls;
  bh.cg_of.assign((size_t)ncls * B, -1);
  bh.dir_local.assign(D, 0);
  std::vector<int> cls_cg0(ncls), cls_ng(ncls);
  for (int c = 0; c < ncls; ++c) {
    const int nd = (int)x.dirs[c].size();
    if (nd > 16) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "brick sweep: %d directions in one octant (at most 16)", nd);
    for (int k = 0; k < nd; ++k) bh.dir_local[x.dirs[c][k]] = k;
    const int ng = (B * nd + kBrickMaxS - 1) / kBrickMaxS;
    int per = (B + ng - 1) / ng;
    while (per * nd > kBrickMaxS) --per;
    if (per > 32) per = 32;
    cls_cg0[c] = (int)bh.cgs.size();
    int ngc = 0;
    for (int b0 = 0; b0 < B; b0 += per, ++ngc) {
      BrickCG g{};
      g.cls = c; g.nd = nd; g.b0 = b0; g.nb = std::min(per, B - b0); g.S = g.nb * nd;
      for (int b = b0; b < b0 + g.nb; ++b) bh.cg_of[(size_t)c * B + b] = (int)bh.cgs.size();
      bh.cgs.push_back(g);
    }
    cls_ng[c] = ngc;
  }

  // ---- per class: positions, flags, rows, closure tables; tasks --------------------------------------------------------------------
  bh.cls.resize(ncls);
  bh.bf_wrow.assign((size_t)ncls * nbf, -1);
  bh.a2pos.assign((size_t)ncls * na, -1);
  std::vector<uint8_t> bf_nord(nbf, 0);
  struct OutEnt { int j, k, ul, vl, wl; };   // an outgoing wall face of a task: entry in Cls::out_*, side, cell
  struct ProtoTask { BrickTask t; int key, cls, J, K, sg; std::vector<OutEnt> outs; int wall_cnt[3]; };
  std::vector<ProtoTask> protos;
  for (int c = 0; c < ncls; ++c) {
    BrickHost::Cls &C = bh.cls[c];
    const int *sg3 = x.sign[c];
    auto ph = [&](int axis, int n, int xp) { return sg3[axis] > 0 ? xp : n - 1 - xp; };  // primed -> physical
    // primed tile / segment intervals
    auto primed_cuts = [&](const std::vector<int> &cut, int n, int axis) {
      std::vector<int> out(cut.size());
      for (size_t k = 0; k < cut.size(); ++k) out[k] = sg3[axis] > 0 ? cut[k] : n - cut[cut.size() - 1 - k];
      return out;
    };
    const std::vector<int> vc = primed_cuts(vcut, nv, x.va), wc = primed_cuts(wcut, nw, x.wa), uc = primed_cuts(ucut, nu, x.pa);
    auto phys_box = [&](int Jp, int Kp, int sp) {
      return box(sg3[x.va] > 0 ? Jp : NTv - 1 - Jp, sg3[x.wa] > 0 ? Kp : NTw - 1 - Kp, sg3[x.pa] > 0 ? sp : nseg - 1 - sp);
    };
    auto actp = [&](int up, int vp, int wp) {  // activity in primed coordinates (outside = inactive)
      if (up < 0 || up >= nu || vp < 0 || vp >= nv || wp < 0 || wp >= nw) return false;
      return x.act[cell_phys(ph(x.pa, nu, up), ph(x.va, nv, vp), ph(x.wa, nw, wp))] != 0;
    };
    const int side_in[3] = {2 * x.pa + (sg3[x.pa] > 0 ? 0 : 1), 2 * x.va + (sg3[x.va] > 0 ? 0 : 1), 2 * x.wa + (sg3[x.wa] > 0 ? 0 : 1)};
    const int side_out[3] = {side_in[0] ^ 1, side_in[1] ^ 1, side_in[2] ^ 1};
    // first pass: which boxes are tasks, their local index
    std::vector<int> task_of((size_t)NTv * NTw * nseg, -1);
    auto pbox = [&](int Jp, int Kp, int sp) { return ((size_t)sp * NTw + Kp) * NTv + Jp; };
    int npos = 0, nrow = 0, nwall = 0;
    const int first_proto = (int)protos.size();
    for (int sp = 0; sp < nseg; ++sp)
      for (int Kp = 0; Kp < NTw; ++Kp)
        for (int Jp = 0; Jp < NTv; ++Jp) {
          if (!box_on[phys_box(Jp, Kp, sp)]) continue;
          ProtoTask P{};
          // earliest start in plane-times: a v- or w-downstream tile runs one plane behind its upstream tile, a u-downstream
          // segment starts when the previous segment has finished
          P.cls = c; P.J = Jp; P.K = Kp; P.sg = sp; P.key = Jp + Kp + uc[sp];
          BrickTask &T = P.t;
          T.nu = uc[sp + 1] - uc[sp]; T.tv = vc[Jp + 1] - vc[Jp]; T.tw = wc[Kp + 1] - wc[Kp];
          T.pos0 = npos; npos += T.nu * kBrickCells;
          T.fu0 = nrow; nrow += kBrickCells;
          T.fv0 = nrow; nrow += T.nu * kBrickTile;
          T.fw0 = nrow; nrow += T.nu * kBrickTile;
          T.ir0 = nrow;  // IRR rows counted below
          T.wo0 = nwall;
          if (T.nu > 64) return nb_fail(h, NANOBTE_E_INVALID, "internal: brick segment of %d planes", T.nu);
          int n_active = 0;
          uint64_t src_planes = 0;
          std::vector<OutEnt> &outs = P.outs;
          int (&wall_cnt)[3] = P.wall_cnt;
          wall_cnt[0] = wall_cnt[1] = wall_cnt[2] = 0;
          // cells in sweep order
          C.th.resize((size_t)npos, 0.0);
          C.qd.resize((size_t)npos, 0.0);
          C.flg.resize((size_t)npos, 0);
          for (int ul = 0; ul < T.nu; ++ul)
            for (int wl = 0; wl < T.tw; ++wl)
              for (int vl = 0; vl < T.tv; ++vl) {
                const int up = uc[sp] + ul, vp = vc[Jp] + vl, wp = wc[Kp] + wl;
                if (!actp(up, vp, wp)) continue;
                const int cphys = cell_phys(ph(x.pa, nu, up), ph(x.va, nv, vp), ph(x.wa, nw, wp));
                const int pos = T.pos0 + ul * kBrickCells + wl * kBrickTile + vl;
                bh.a2pos[(size_t)c * na + x.G->cell2act[cphys]] = pos;
                uint8_t f = BRK_ACT;
                ++n_active;
                const bool upact[3] = {actp(up - 1, vp, wp), actp(up, vp - 1, wp), actp(up, vp, wp - 1)};
                const int loc[3] = {ul, vl, wl};
                const uint8_t inj[3] = {BRK_INJ_U, BRK_INJ_V, BRK_INJ_W};
                for (int k = 0; k < 3; ++k) {
                  if (upact[k] && loc[k] > 0) continue;  // interior neighbour inside the task: plane buffer / registers
                  int row;
                  if (loc[k] == 0) row = k == 0 ? T.fu0 + wl * kBrickTile + vl : k == 1 ? T.fv0 + ul * kBrickTile + wl : T.fw0 + ul * kBrickTile + vl;
                  else { row = nrow++; f |= inj[k]; }
                  if (!upact[k]) {  // a wall: the closure kernel owns this row
                    const int bf = x.facebf[(size_t)cphys * 6 + side_in[k]];
                    if (bf < 0) return nb_fail(h, NANOBTE_E_INVALID, "internal: brick inflow face of cell %d missing", cphys);
                    C.in_row.push_back(row);
                    C.in_bf.push_back(bf);
                  }
                }
                bool wallout = false;
                const bool dnact[3] = {actp(up + 1, vp, wp), actp(up, vp + 1, wp), actp(up, vp, wp + 1)};
                for (int k = 0; k < 3; ++k)
                  if (!dnact[k]) {
                    const int bf = x.facebf[(size_t)cphys * 6 + side_out[k]];
                    if (bf < 0) return nb_fail(h, NANOBTE_E_INVALID, "internal: brick outflow face of cell %d missing", cphys);
                    wallout = true;
                    outs.push_back({(int)C.out_bf.size(), k, ul, vl, wl});
                    ++wall_cnt[k];
                    C.out_bf.push_back(bf);
                    C.out_row.push_back(nwall);
                    C.out_ord.push_back(bf_nord[bf]++);
                    bh.bf_wrow[(size_t)c * nbf + bf] = nwall;
                  }
                if (wallout) { f |= BRK_WALL; ++nwall; }
                const double q = x.Qdot ? x.Qdot[cphys] : 0.0;
                if (q != 0.0) { f |= BRK_SRC; src_planes |= 1ull << ul; }
                C.flg[pos] = f;
                C.th[pos] = x.T_init ? x.T_init[cphys] - x.T_ref : 0.0;
                C.qd[pos] = q;
              }
          T.plain = n_active == T.nu * T.tv * T.tw;
          T.src_lo = (uint32_t)src_planes; T.src_hi = (uint32_t)(src_planes >> 32);
          T.wall_any = nwall > T.wo0;
          T.wu0 = T.wv0 = T.ww0 = -1;
          // A fully active box whose downstream faces are each all wall (and then without a downstream tile) or all interior:
          // its wall rows become face blocks with the addressing of the inflow faces (u-face [w][v], v-face [u][w], w-face
          // [u][v]), so that the sweep stores wall values where it would store the face of a downstream tile -- no pass over
          // the wall cells afterwards.
          auto box_exists = [&](int Jq, int Kq, int sq) {
            return Jq >= 0 && Jq < NTv && Kq >= 0 && Kq < NTw && sq >= 0 && sq < nseg && box_on[phys_box(Jq, Kq, sq)] != 0;
          };
          const int face_n[3] = {T.tv * T.tw, T.nu * T.tw, T.nu * T.tv};
          const bool dn_exists[3] = {box_exists(Jp, Kp, sp + 1), box_exists(Jp + 1, Kp, sp), box_exists(Jp, Kp + 1, sp)};
          bool pure = T.plain && T.wall_any;
          for (int k = 0; k < 3; ++k) pure = pure && (wall_cnt[k] == 0 || (wall_cnt[k] == face_n[k] && !dn_exists[k]));
          if (pure) {
            nwall = T.wo0;  // the rows given out cell by cell above are taken back
            if (wall_cnt[0]) { T.wu0 = nwall; nwall += kBrickCells; }
            if (wall_cnt[1]) { T.wv0 = nwall; nwall += T.nu * kBrickTile; }
            if (wall_cnt[2]) { T.ww0 = nwall; nwall += T.nu * kBrickTile; }
            for (const OutEnt &e : outs) {
              const int row = e.k == 0 ? T.wu0 + e.wl * kBrickTile + e.vl : e.k == 1 ? T.wv0 + e.ul * kBrickTile + e.wl : T.ww0 + e.ul * kBrickTile + e.vl;
              C.out_row[e.j] = row;
              bh.bf_wrow[(size_t)c * nbf + C.out_bf[e.j]] = row;
            }
            T.wall_any = 0;  // nothing left for the pass over the wall cells
          }
          outs.clear();
          outs.shrink_to_fit();
          task_of[pbox(Jp, Kp, sp)] = (int)protos.size();
          protos.push_back(P);
        }
    // links (indices into protos for now)
    for (int k = first_proto; k < (int)protos.size(); ++k) {
      ProtoTask &P = protos[k];
      auto at = [&](int Jp, int Kp, int sp) {
        if (Jp < 0 || Jp >= NTv || Kp < 0 || Kp >= NTw || sp < 0 || sp >= nseg) return -1;
        return task_of[pbox(Jp, Kp, sp)];
      };
      P.t.up_u = at(P.J, P.K, P.sg - 1);
      P.t.up_v = at(P.J - 1, P.K, P.sg);
      P.t.up_w = at(P.J, P.K - 1, P.sg);
      // face modes: TAGGED if every upstream cell across the face is active (then every row of the face is the upstream
      // task's), COUNTER if the face mixes task rows and closure rows
      auto face_mode = [&](int up, bool vface) {
        if (up < 0) return (int32_t)BRK_FACE_BOUNDARY;
        const int n2 = vface ? P.t.tw : P.t.tv;
        for (int ul = 0; ul < P.t.nu; ++ul)
          for (int k = 0; k < n2; ++k) {
            const int upp = uc[P.sg] + ul, vp = vface ? vc[P.J] - 1 : vc[P.J] + k, wp = vface ? wc[P.K] + k : wc[P.K] - 1;
            if (!actp(upp, vp, wp)) return (int32_t)BRK_FACE_COUNTER;
          }
        return (int32_t)BRK_FACE_TAGGED;
      };
      P.t.fv_mode = face_mode(P.t.up_v, true);
      P.t.fw_mode = face_mode(P.t.up_w, false);
      if (P.t.fv_mode == BRK_FACE_COUNTER) protos[P.t.up_v].t.publish = 1;
      if (P.t.fw_mode == BRK_FACE_COUNTER) protos[P.t.up_w].t.publish = 1;
      const int du = at(P.J, P.K, P.sg + 1), dv = at(P.J + 1, P.K, P.sg), dw = at(P.J, P.K + 1, P.sg);
      P.t.dn_fu0 = du >= 0 ? protos[du].t.fu0 : -1;
      P.t.dn_fv0 = dv >= 0 ? protos[dv].t.fv0 : -1;
      P.t.dn_fw0 = dw >= 0 ? protos[dw].t.fw0 : -1;

    }
    C.scratch_row = nrow; nrow += kBrickTile;
    C.npos = npos; C.nrow = nrow; C.nwall = std::max(1, nwall);
    C.th.resize((size_t)npos + 64, 0.0);
    C.qd.resize((size_t)npos + 64, 0.0);
    C.flg.resize((size_t)npos + 64, 0);
  }
  bh.bf_nord = bf_nord;

  // ---- records of the fast inflow kernel: per inflow row its face, type, the mirror class and the wall row the specular part
  // comes from; per class the (at most 8) permutations "direction -> mirrored direction" that occur ---------------------------------
  {
    std::vector<int> dcls(D, 0);
    for (int c = 0; c < ncls; ++c)
      for (int d : x.dirs[c]) dcls[d] = c;
    bh.in_perm.assign((size_t)ncls * 8 * 16, 255);
    bh.in_fast = true;
    for (int c = 0; c < ncls && bh.in_fast; ++c) {
      BrickHost::Cls &C = bh.cls[c];
      const int nd = (int)x.dirs[c].size();
      int nperm = 0;
      C.in_rec.resize(C.in_row.size());
      for (size_t k = 0; k < C.in_row.size() && bh.in_fast; ++k) {
        BrickInRow R{};
        R.bf = C.in_bf[k]; R.row = C.in_row[k]; R.msrc = -1; R.type = (uint8_t)x.G->bf_type[R.bf]; R.cm = 0; R.perm = 0;
        if (R.type == NANOBTE_SPECULAR || R.type == NANOBTE_MIXED) {
          uint8_t pm[16];
          int cm = -1;
          for (int dl = 0; dl < 16; ++dl) pm[dl] = 255;
          for (int dl = 0; dl < nd; ++dl) {
            const int md = x.G->bf_mirror[(size_t)R.bf * D + x.dirs[c][dl]];
            if (md < 0) continue;
            if (cm >= 0 && dcls[md] != cm) bh.in_fast = false;  // the mirror images of one class in two classes: general kernel
            cm = dcls[md];
            pm[dl] = (uint8_t)bh.dir_local[md];
          }
          if (cm >= 0) {
            R.cm = (uint8_t)cm;
            R.msrc = bh.bf_wrow[(size_t)cm * nbf + R.bf];
            if (R.msrc < 0) bh.in_fast = false;
            int id = -1;
            for (int q = 0; q < nperm && id < 0; ++q)
              if (std::equal(pm, pm + 16, &bh.in_perm[((size_t)c * 8 + q) * 16])) id = q;
            if (id < 0) {
              if (nperm == 8) { bh.in_fast = false; break; }
              id = nperm++;
              std::copy(pm, pm + 16, &bh.in_perm[((size_t)c * 8 + id) * 16]);
            }
            R.perm = (uint8_t)id;
          }
        }
        C.in_rec[k] = R;
      }
      // the fast kernel takes kBrickInRows records at a time and branches once per batch: the records go by type (thermalizing
      // rows never change after the first launch and are left out), every type padded to whole batches with empty records
      std::vector<BrickInRow> by_type;
      for (int ty : {NANOBTE_DIFFUSE, NANOBTE_SPECULAR, NANOBTE_MIXED}) {
        for (const BrickInRow &R : C.in_rec)
          if (R.type == ty) by_type.push_back(R);
        while (by_type.size() % kBrickInRows) {
          BrickInRow E{};
          E.bf = -1; E.row = 0; E.msrc = -1; E.type = (uint8_t)ty;
          by_type.push_back(E);
        }
      }
      C.in_rec.swap(by_type);
    }
    bh.cg0.assign(cls_cg0.begin(), cls_cg0.end());
    for (int c = 0; c < ncls; ++c) {  // records of the gsum kernel (the wall rows are final here)
      BrickHost::Cls &C = bh.cls[c];
      C.out_rec.resize(C.out_bf.size());
      for (size_t j = 0; j < C.out_rec.size(); ++j) {
        BrickOutRow R{};
        R.bf = C.out_bf[j]; R.row = C.out_row[j]; R.ord = C.out_ord[j]; R.type = (uint8_t)x.G->bf_type[R.bf];
        C.out_rec[j] = R;
      }
    }
    for (int c = 1; c < ncls; ++c)  // the same band groups in every class (then the mirror group is the same group index)
      if (cls_ng[c] != cls_ng[0] || x.dirs[c].size() != x.dirs[0].size()) bh.in_fast = false;
  }

  // ---- tasks: one per (proto, group), topological launch order ----------------------------------------------------------------------
  // key = primed tile/segment diagonal: every upstream task has a smaller key.  Within a key the classes and groups
  // are interleaved so that all octants advance together.
  std::vector<int> order(protos.size());
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int p, int q) { return protos[p].key < protos[q].key; });
  std::vector<int> first_task(protos.size(), -1);
  int ng_max = 0;
  for (int c = 0; c < ncls; ++c) ng_max = std::max(ng_max, cls_ng[c]);
  // tasks of one proto are consecutive per group ROUND: (key, group, proto) order keeps the groups of a class abreast
  std::vector<std::vector<int>> task_id(ng_max, std::vector<int>(protos.size(), -1));
  {
    size_t lo = 0;
    while (lo < order.size()) {
      size_t hi = lo;
      while (hi < order.size() && protos[order[hi]].key == protos[order[lo]].key) ++hi;
      for (int g = 0; g < ng_max; ++g)
        for (size_t k = lo; k < hi; ++k) {
          const ProtoTask &P = protos[order[k]];
          if (g >= cls_ng[P.cls]) continue;
          BrickTask T = P.t;
          T.cg = cls_cg0[P.cls] + g;
          task_id[g][order[k]] = (int)bh.tasks.size();
          bh.tasks.push_back(T);
        }
      lo = hi;
    }
  }
  for (BrickTask &T : bh.tasks) {  // proto indices -> task ids of the same group
    const int g = T.cg - cls_cg0[bh.cgs[T.cg].cls];
    if (T.up_u >= 0) T.up_u = task_id[g][T.up_u];
    if (T.up_v >= 0) T.up_v = task_id[g][T.up_v];
    if (T.up_w >= 0) T.up_w = task_id[g][T.up_w];
  }
  for (size_t k = 0; k < bh.tasks.size(); ++k) {
    const BrickTask &T = bh.tasks[k];
    if (T.up_u >= (int)k || T.up_v >= (int)k || T.up_w >= (int)k) return nb_fail(h, NANOBTE_E_INVALID, "internal: brick task order is not topological");
  }

  // ---- blocks of every (class, group) and the coefficient blocks ---------------------------------------------------------------------
  int64_t inf = 0, wall = 0, part = 0, e = 0, cf = 0;
  for (BrickCG &g : bh.cgs) {
    const BrickHost::Cls &C = bh.cls[g.cls];
    auto pad = [](int64_t v) { return (v + 31) / 32 * 32; };
    g.inf_base = inf; inf = pad(inf + (int64_t)C.nrow * kBrickRow);
    g.wall_base = wall; wall = pad(wall + (int64_t)C.nwall * kBrickRow);
    g.part_base = part; part = pad(part + (int64_t)5 * C.npos);
    g.e_base = e; e = pad(e + (int64_t)C.npos * g.S);  // the stored distribution: pitch S (it is the big array)
    g.coef_base = cf;
    for (int bl = 0; bl < g.nb; ++bl)
      for (int dl = 0; dl < g.nd; ++dl) {
        const size_t row = (size_t)x.cls_row0[g.cls] + (size_t)dl * B + (g.b0 + bl);
        for (int k = 0; k < 5; ++k) bh.coef.push_back(x.coef[row * 8 + k]);
      }
    // the loop above is band-major: system = band_local * nd + dir_local
    for (int dl = 0; dl < g.nd; ++dl) {
      const int d = x.dirs[g.cls][dl];
      bh.coef.push_back(x.cm->w[d]);
      for (int k = 0; k < 3; ++k) bh.coef.push_back(x.cm->w[d] * x.cm->s[3 * (size_t)d + k]);
    }
    for (int bl = 0; bl < g.nb; ++bl) {
      bh.coef.push_back(1.0 / x.cm->tau[g.b0 + bl]);
      bh.coef.push_back(x.cm->v[g.b0 + bl]);
    }
    while (bh.coef.size() & 3) bh.coef.push_back(0.0);
    cf = (int64_t)bh.coef.size();
  }
  bh.inf_total = inf; bh.wall_total = wall; bh.part_total = part; bh.e_total = e;
  return 0;
}

int nb_brick_upload(nanobte_solver *h, Arena &A, BrickHost &bh) {
  if (!h->brick) h->brick = new BrickState();
  BrickState &bs = *h->brick;
  BrickArgs &a = bs.a;
  a.tasks = A.put(bh.tasks);
  a.cgs = A.put(bh.cgs);
  a.n_tasks = (int)bh.tasks.size();
  for (int c = 0; c < bh.ncls; ++c) {
    BrickHost::Cls &C = bh.cls[c];
    bs.th[c] = A.put(C.th);
    a.th[c] = bs.th[c];
    a.qd[c] = A.put(C.qd);
    a.flg[c] = A.put(C.flg);
    a.npos[c] = C.npos;
    a.scratch_row[c] = C.scratch_row;
    bs.in_row[c] = A.put(C.in_row);
    bs.in_bf[c] = A.put(C.in_bf);
    bs.n_in[c] = (int32_t)C.in_row.size();
    bs.out_bf[c] = A.put(C.out_bf);
    bs.out_row[c] = A.put(C.out_row);
    bs.out_ord[c] = A.put(C.out_ord);
    bs.out_rec[c] = A.put(C.out_rec);
    bs.n_out[c] = (int32_t)C.out_bf.size();
    if (bh.in_fast) { bs.in_rec[c] = A.put(C.in_rec); bs.n_rec[c] = (int32_t)C.in_rec.size(); }
    bs.cg0[c] = bh.cg0[c];
  }
  a.inf = A.zeros<double>((size_t)bh.inf_total);
  a.wall = A.zeros<double>((size_t)bh.wall_total);
  a.part = A.zeros<double>((size_t)bh.part_total);
  a.e = A.zeros<double>((size_t)bh.e_total);
  a.coef = A.put(bh.coef);
  unsigned int *sync = A.zeros<unsigned int>((size_t)a.n_tasks + 1);
  a.ticket = sync;
  a.prog = sync + 1;
  bs.bf_wrow = A.put(bh.bf_wrow);
  bs.dir_local = A.put(bh.dir_local);
  bs.cg_of = A.put(bh.cg_of);
  bs.a2pos = A.put(bh.a2pos);
  {
    const int na = (int)(bh.a2pos.size() / bh.ncls);
    std::vector<int32_t> pos2a((size_t)bh.cls[0].npos + 64, -1);
    for (int a = 0; a < na; ++a) pos2a[bh.a2pos[a]] = a;
    bs.pos2a = A.put(pos2a);
  }
  bs.bf_nord = A.put(bh.bf_nord);
  bs.in_perm = A.put(bh.in_perm);
  bs.in_fast = bh.in_fast && std::getenv("NANOBTE_BRICK_SLOW_INFLOW") == nullptr;
  if (!A.dry && !h->aux_stream && std::getenv("NANOBTE_NO_AUX_STREAM") == nullptr) {
    if (cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess)
      return nb_fail(h, NANOBTE_E_CUDA, "second stream of the tile-dataflow path");
  }
  bs.n_cg = (int)bh.cgs.size();
  bs.smem = nb_brick_smem_bytes();
  bs.grid = std::max(1, std::min(a.n_tasks, 3 * h->n_sm));
  bs.inf_total = bh.inf_total; bs.wall_total = bh.wall_total; bs.part_total = bh.part_total; bs.e_total = bh.e_total;
  bs.s_max = 0;
  for (const BrickCG &g : bh.cgs) bs.s_max = std::max(bs.s_max, g.S);
  return A.rc;
}
