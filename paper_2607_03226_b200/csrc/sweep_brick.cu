// sweep_brick.cu -- (a2)+(a4)+(a6) fused: tile-dataflow transport sweep with the moment reduction inside
// (SURVEY 8.f row f1).  See brick.h for the decomposition and the row spaces.
//
// Per update (Eq. 4, 91 Eq. 11, 104/110, 178; first-order upwind R1; uniform spacing):
//   eps_c = k_th th_c + k_Q Qdot_c + c_u eps_up,u + c_v eps_up,v + c_w eps_up,w          (coefficients pre-divided by
//   1/tau_b + v_b sum_a |s_a|/h_a, as in sweep_structured.cu)
// and per cell and u-plane the partial moments of the task's systems (Eq. 5, R13, Eq. 7):
//   part0 = sum w/tau eps, part1 = sum w eps, part2..4 = sum v w s eps.
//
// One u-plane of a task in two roles:
//   substitution  thread = system.  Tasks whose box is fully active (BrickTask::plain; with tile cuts that follow the
//                 mask that is every task of a box-shaped geometry) run branch-free, software-pipelined code with the tile
//                 width and the row count as template constants (fast_plane): per cell one LDS (u-upwind), one STS,
//                 4 fp64 operations.  Planes with a source or a stored distribution take plain_plane, other tasks the
//                 per-cell path that reads the flag bytes (walls inside the tile).
//   moments       thread = one cell x half of the class's directions, all bands: the band sums first (3 fp64 operations
//                 per value), the direction weights once per plane; a warp owns 16 cells, one shuffle joins the halves.
// Tile faces cross CTAs through L2 tagged with the sweep parity (brick.h, BRK_FACE_TAGGED): no fence, no counter.
// Shared memory is the scarce resource (128 B/clk per SM against 64 DFMA/clk; a broadcast load still returns 8 B per
// lane): per update STS 8 B + u-upwind 8 B + theta 8 B + moments 8 B + band coefficients ~3 B = 35 B.
#include <algorithm>

#include "brick.h"

namespace {

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int *p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(unsigned int *p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Progress of the two upstream tiles (v: lane 0, w: lane 1 of every warp), polled with ONE acquire load for both and
// remembered: an upstream tile that started earlier is usually many planes ahead, and then no poll is needed at all.
// The published rows are read with L2 loads (ld.cg); __syncwarp orders the other lanes behind the polling lanes.
struct Upstream {
  const unsigned int *pv, *pw;  // progress words (nullptr: no upstream task -- boundary rows, always there)
  unsigned int seen_v, seen_w;
  __device__ __forceinline__ void init(const unsigned int *prog, int up_v, int up_w) {  // < 0: nothing to wait for
    pv = up_v >= 0 ? prog + up_v : nullptr;
    pw = up_w >= 0 ? prog + up_w : nullptr;
    seen_v = pv ? 0u : 0x7fffffffu;
    seen_w = pw ? 0u : 0x7fffffffu;
  }
  __device__ __forceinline__ bool poll(unsigned int need) {  // true in every lane if both have published `need` planes
    if (seen_v >= need && seen_w >= need) return true;
    const int lane = threadIdx.x & 31;
    const unsigned int *p = lane == 0 ? pv : pw;
    unsigned int v = 0x7fffffffu;
    if (lane < 2 && p) v = ld_acquire(p);
    seen_v = __shfl_sync(0xffffffffu, v, 0);
    seen_w = __shfl_sync(0xffffffffu, v, 1);
    return seen_v >= need && seen_w >= need;
  }
  __device__ __forceinline__ void wait(unsigned int need) {
    while (!poll(need)) __nanosleep(20);
  }
};

__device__ __forceinline__ void wait_progress(const unsigned int *prog, int up, unsigned int need) {
  if (up >= 0) {
    if ((threadIdx.x & 31) == 0) {
      while (ld_acquire(prog + up) < need) __nanosleep(40);
    }
    __syncwarp();
  }
}

constexpr int kP = kBrickPitch;

// A value that crosses a tile face: its least significant mantissa bit is the sweep parity (brick.h, BRK_FACE_TAGGED).
__device__ __forceinline__ double tag(double x, unsigned par) {
  return __hiloint2double(__double2hiint(x), (int)(((unsigned)__double2loint(x) & ~1u) | par));
}
// Face rows are read at the L2 (the point of coherence), and every time the code says so (the settle loop re-reads them).
__device__ __forceinline__ double ld_face(const double *p) {
  double v;
  asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned stale_bit(double x, unsigned par) { return ((unsigned)__double2loint(x) ^ par) & 1u; }

#ifdef BRICK_PROF
__device__ unsigned long long g_brick_prof[16];
constexpr int kBrickTlMax = 1 << 15;
__device__ unsigned long long g_brick_tl[kBrickTlMax][4];  // per task: ticket taken, first plane ready, done [ns]; SM | nu << 32
__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long v;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(v));
  return v;
}
#define PROF_T(var) const long long var = clock64()
#define PROF_ADD(k, a, b) if (t == 0) prof[k] += (unsigned long long)((b) - (a))
#else
#define PROF_T(var)
#define PROF_ADD(k, a, b)
#endif

struct BrickSmem {
  double plane[kBrickCells * kBrickPitch];     // [cell][system]: eps of the previous u-plane (u-upwind values)
  double th[kBrickCells];                      // theta of the plane's cells
  double qd[kBrickCells];                      // Qdot
  unsigned long long flg[2][kBrickCells / 8];  // flag bytes, one 64-bit word per row of 8 cells, two stages
  double dcoef[16 * 4];                        // [nd][4]  w, w sx, w sy, w sz
  double bcoef[32 * 2];                        // [nb][2]  1/tau, v
  int task;
};
static_assert(3 * (sizeof(BrickSmem) + 1024) <= 228 * 1024, "three CTAs per SM");

struct Sys {           // what a substitution thread keeps for its system
  double k_th, k_Q, c_u, c_v, c_w;
};

// ---- one u-plane of a fully active box, TV cells per row: straight-line code ---------------------------------------------------------
// pl = plane buffer + system; ew[v] = w-upwind values (in: tile-face inflow, out: last row); inv[w] = v-face inflow of row w;
// dn_fv_u / eout_u = this plane's rows of the v-downstream tile / of the stored distribution (pitch S; nullptr: none).
template <int TV>
__device__ __forceinline__ void plain_plane(double *__restrict__ pl, const double *__restrict__ th, const double *__restrict__ qd,
                                            const Sys &c, const int tw, const bool src, double (&ew)[kBrickTile],
                                            const double (&inv)[kBrickTile], double *dn_fv_u, double *eout_u, const int S,
                                            const unsigned par) {
#pragma unroll
  for (int w = 0; w < kBrickTile; ++w) {
    if (w < tw) {
      double *row = pl + w * kBrickTile * kP;
      double r[TV], eu[TV];
#pragma unroll
      for (int v = 0; v < TV; ++v) eu[v] = row[v * kP];
#pragma unroll
      for (int v = 0; v < TV; v += 2) {
        const double2 t2 = *reinterpret_cast<const double2 *>(th + w * kBrickTile + v);
        r[v] = c.k_th * t2.x;
        if (v + 1 < TV) r[v + 1] = c.k_th * t2.y;
      }
      if (src) {
#pragma unroll
        for (int v = 0; v < TV; v += 2) {
          const double2 q2 = *reinterpret_cast<const double2 *>(qd + w * kBrickTile + v);
          r[v] = fma(c.k_Q, q2.x, r[v]);
          if (v + 1 < TV) r[v + 1] = fma(c.k_Q, q2.y, r[v + 1]);
        }
      }
#pragma unroll
      for (int v = 0; v < TV; ++v) r[v] = fma(c.c_w, ew[v], fma(c.c_u, eu[v], r[v]));  // same association as fast_plane
      double ev = inv[w];
#pragma unroll
      for (int v = 0; v < TV; ++v) {
        ev = fma(c.c_v, ev, r[v]);  // the v-chain is the only dependency between the cells of a row
        ew[v] = ev;
        row[v * kP] = ev;
      }
      if (dn_fv_u) dn_fv_u[w * kBrickRow] = tag(ev, par);
      if (eout_u) {
#pragma unroll
        for (int v = 0; v < TV; ++v) __stcs(eout_u + (w * kBrickTile + v) * S, ew[v]);
      }
    }
  }
}

// ---- the same without a branch: no source in the plane, the distribution not stored, the v-face rows always written (tiles on
// the boundary write a scratch row), ROWS = 7 or 8 rows computed (rows >= tw of a shorter tile work on values nobody reads).  Written
// software-pipelined: the loads and the chain-independent half of row w+1 sit between the chain steps of row w, so that a warp
// has work of its own during the 8-cycle DFMA latency of the v-chain.
template <int TV, int ROWS>
__device__ __forceinline__ void fast_plane(double *__restrict__ pl, const double *__restrict__ th, const Sys &c,
                                           double (&ew)[kBrickTile], const double (&inv)[kBrickTile], double *__restrict__ dn_fv_u,
                                           const unsigned par) {
  double rp[TV], rn[TV];
  {
    double eu[TV];
#pragma unroll
    for (int v = 0; v < TV; ++v) eu[v] = pl[v * kP];
#pragma unroll
    for (int v = 0; v < TV; v += 2) {
      const double2 t2 = *reinterpret_cast<const double2 *>(th + v);
      rp[v] = fma(c.c_u, eu[v], c.k_th * t2.x);
      if (v + 1 < TV) rp[v + 1] = fma(c.c_u, eu[v + 1], c.k_th * t2.y);
    }
  }
#pragma unroll
  for (int w = 0; w < ROWS; ++w) {
    double *row = pl + w * kBrickTile * kP;
    double eu[TV], tn[TV];
    if (w + 1 < ROWS) {
#pragma unroll
      for (int v = 0; v < TV; ++v) eu[v] = row[(kBrickTile + v) * kP];
#pragma unroll
      for (int v = 0; v < TV; v += 2) {
        const double2 t2 = *reinterpret_cast<const double2 *>(th + (w + 1) * kBrickTile + v);
        tn[v] = t2.x;
        if (v + 1 < TV) tn[v + 1] = t2.y;
      }
    }
    double ev = inv[w];
#pragma unroll
    for (int v = 0; v < TV; ++v) {
      ev = fma(c.c_v, ev, fma(c.c_w, ew[v], rp[v]));  // the v-chain is the only dependency between the cells of a row
      ew[v] = ev;
      row[v * kP] = ev;
      if (w + 1 < ROWS) rn[v] = fma(c.c_u, eu[v], c.k_th * tn[v]);
    }
    dn_fv_u[w * kBrickRow] = tag(ev, par);
#pragma unroll
    for (int v = 0; v < TV; ++v) rp[v] = rn[v];
  }
}

// ---- moments of one u-plane, one thread: one cell, ND consecutive directions, all bands ---------------------------------------------------
// The band sums come first (three weights: 1/tau_b, 1, v_b -- 3 fp64 operations per value), the direction weights once per
// plane:  m0 = sum_d w_d sum_b eps/tau_b,  m1 = sum_d w_d sum_b eps,  m2..4 = sum_d w_d s_d sum_b v_b eps.
// row = plane buffer + cell * pitch + first direction; bcoef = [nb][2] (1/tau, v); dcoef = [ND][4] (w, w sx, w sy, w sz).
template <int ND>
__device__ __forceinline__ void moments_cell(const double *__restrict__ row, const double *__restrict__ bcoef,
                                             const double *__restrict__ dcoef, const int nb, const int nd, double (&m)[5]) {
  double A[ND], Bs[ND], Cv[ND];
#pragma unroll
  for (int j = 0; j < ND; ++j) A[j] = Bs[j] = Cv[j] = 0.0;
#pragma unroll 2
  for (int b = 0; b < nb; ++b) {
    const double2 bc = *reinterpret_cast<const double2 *>(bcoef + 2 * b);
#pragma unroll
    for (int j = 0; j < ND; ++j) {
      const double e = row[j];
      A[j] = fma(bc.x, e, A[j]);
      Bs[j] += e;
      Cv[j] = fma(bc.y, e, Cv[j]);
    }
    row += nd;
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) m[k] = 0.0;
#pragma unroll
  for (int j = 0; j < ND; ++j) {
    const double2 c01 = *reinterpret_cast<const double2 *>(dcoef + 4 * j);
    const double2 c23 = *reinterpret_cast<const double2 *>(dcoef + 4 * j + 2);
    m[0] = fma(c01.x, A[j], m[0]);
    m[1] = fma(c01.x, Bs[j], m[1]);
    m[2] = fma(c01.y, Cv[j], m[2]);
    m[3] = fma(c23.x, Cv[j], m[3]);
    m[4] = fma(c23.y, Cv[j], m[4]);
  }
}

__global__ void __launch_bounds__(kBrickMaxS, 3) sweep_brick_kernel(const BrickArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  BrickSmem &sm = *reinterpret_cast<BrickSmem *>(smem_raw);
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;

  for (;;) {
    __syncthreads();  // the previous task's shared memory is dead
    if (t == 0) sm.task = (int)atomicAdd(a.ticket, 1u);
    __syncthreads();
    const int task = sm.task;
    if (task >= a.n_tasks) break;
#ifdef BRICK_PROF
    const unsigned long long tl0 = gtime();
#endif
    const BrickTask T = a.tasks[task];
    const BrickCG G = a.cgs[T.cg];
    const int S = G.S;
    const bool on = t < S;              // this thread owns system t of the group
    const int s = on ? t : 0;
    const double *th_g = a.th[G.cls] + T.pos0, *qd_g = a.qd[G.cls] + T.pos0;
    const uint8_t *flg_g = a.flg[G.cls] + T.pos0;
    double *inf = a.inf + G.inf_base + s;
    double *wall = a.wall + G.wall_base + (int64_t)T.wo0 * kBrickRow + s;
    double *part = a.part + G.part_base + T.pos0;
    const int64_t npos = a.npos[G.cls];
    double *eout = a.store_e ? a.e + G.e_base + (int64_t)T.pos0 * S + s : nullptr;  // pitch S
    const double *irr = inf + (int64_t)T.ir0 * kBrickRow;
    const double *fv = inf + (int64_t)T.fv0 * kBrickRow, *fw = inf + (int64_t)T.fw0 * kBrickRow;
    double *dn_fu = T.dn_fu0 >= 0 ? inf + (int64_t)T.dn_fu0 * kBrickRow : nullptr;
    double *dn_fv = T.dn_fv0 >= 0 ? inf + (int64_t)T.dn_fv0 * kBrickRow : nullptr;
    double *dn_fw = T.dn_fw0 >= 0 ? inf + (int64_t)T.dn_fw0 * kBrickRow : nullptr;
    // a face that is all wall (and has no downstream tile): its values go to the task's wall rows, which have the same
    // addressing as a downstream tile's face rows (setup_brick.cu) -- the closures read them there
    if (T.wu0 >= 0) dn_fu = a.wall + G.wall_base + (int64_t)T.wu0 * kBrickRow + s;
    if (T.wv0 >= 0) dn_fv = a.wall + G.wall_base + (int64_t)T.wv0 * kBrickRow + s;
    if (T.ww0 >= 0) dn_fw = a.wall + G.wall_base + (int64_t)T.ww0 * kBrickRow + s;
    const unsigned long long src_planes = ((unsigned long long)T.src_hi << 32) | T.src_lo;
    const bool plain = T.plain && T.tv >= 4;
    const bool rows7 = T.tw <= 7;  // the branch-free substitution computes 7 or 8 rows
    double *scratch = a.inf + G.inf_base + (int64_t)a.scratch_row[G.cls] * kBrickRow + s;  // 8 rows nobody reads

    // coefficients of this thread's system; moment tables of the group
    const double *cf = a.coef + G.coef_base;
    Sys c;
    c.k_th = cf[s * 5 + 0]; c.k_Q = cf[s * 5 + 1]; c.c_u = cf[s * 5 + 2]; c.c_v = cf[s * 5 + 3]; c.c_w = cf[s * 5 + 4];
    if (t < G.nd * 4) sm.dcoef[t] = cf[S * 5 + t];
    if (t < G.nb * 2) sm.bcoef[t] = cf[S * 5 + G.nd * 4 + t];

    // stage the cell tables of a plane: theta 32 x 16 B, Qdot 32 x 16 B, flags 4 x 16 B
    auto stage = [&](int un) {
      const int64_t off = (int64_t)un * kBrickCells;
      if (t < 32) cp_async16(&sm.th[2 * t], th_g + off + 2 * t);
      else if (t < 64) cp_async16(&sm.qd[2 * (t - 32)], qd_g + off + 2 * (t - 32));
      else if (t < 68) cp_async16(reinterpret_cast<unsigned char *>(sm.flg[un & 1]) + 16 * (t - 64), flg_g + off + 16 * (t - 64));
    };
    stage(0);
    // u-face inflow -> plane buffer (the previous segment of the pencils, or boundary values)
    wait_progress(a.prog, T.up_u, 0x7fffffffu);
    if (on) {
      const double *fu = inf + (int64_t)T.fu0 * kBrickRow;
#pragma unroll 8
      for (int cc = 0; cc < kBrickCells; ++cc) sm.plane[cc * kP + s] = __ldcg(fu + cc * kBrickRow);
    }
    // v- and w-face inflow of plane 0
    const unsigned par = a.parity;
#ifdef BRICK_PROF
    unsigned long long prof[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#endif
    Upstream ups;  // only the faces that mix task rows and closure rows are followed through counters
    ups.init(a.prog, T.fv_mode == BRK_FACE_COUNTER ? T.up_v : -1, T.fw_mode == BRK_FACE_COUNTER ? T.up_w : -1);
    const bool counters = T.fv_mode == BRK_FACE_COUNTER || T.fw_mode == BRK_FACE_COUNTER;
    const int chk_v = T.fv_mode == BRK_FACE_TAGGED ? T.tw : 0, chk_w = T.fw_mode == BRK_FACE_TAGGED ? T.tv : 0;
    double ew[kBrickTile], inv[kBrickTile];
    auto load_faces = [&]() {  // fv / fw point at the rows of the plane to come
#pragma unroll
      for (int k = 0; k < kBrickTile; ++k) {
        inv[k] = on ? ld_face(fv + k * kBrickRow) : 0.0;
        ew[k] = on ? ld_face(fw + k * kBrickRow) : 0.0;
      }
    };
    // tagged faces: rows that still carry the other parity are last sweep's -- load again until the upstream tile has
    // written them (every thread follows its own system; nobody else's values are involved)
    auto settle_faces = [&]() {
      if (on && (chk_v | chk_w)) {
        for (;;) {
          unsigned bad = 0;
#pragma unroll
          for (int k = 0; k < kBrickTile; ++k) {
            if (k < chk_v) bad |= stale_bit(inv[k], par);
            if (k < chk_w) bad |= stale_bit(ew[k], par);
          }
          if (!bad) break;
#ifdef BRICK_PROF
          if (t == 0) prof[7] += 1;
#endif
          __nanosleep(20);
          load_faces();
        }
      }
      fv += kBrickTile * kBrickRow;
      fw += kBrickTile * kBrickRow;
    };
    if (counters) ups.wait(1u);
    load_faces();
    settle_faces();
    cp_async_wait_all();
    __syncthreads();
#ifdef BRICK_PROF
    const unsigned long long tl1 = gtime();
#endif

    const int nd = G.nd;

    int ip = 0;  // next row of the IRR stream (same value in every thread)
    for (int u = 0; u < T.nu; ++u) {
      PROF_T(p0);
      const int st = u & 1;
      const bool last_u = u + 1 == T.nu;
      // ------------------------------------------ substitution: thread = system ------------------------------------------
      if (on) {
        double *pl = sm.plane + s;
        if (plain) {
          const bool src = (src_planes >> u) & 1ull;
          if (!src && !eout) {
            double *dfv = dn_fv ? dn_fv : scratch;
            switch (T.tv) {
              case 8: if (rows7) fast_plane<8, 7>(pl, sm.th, c, ew, inv, dfv, par); else fast_plane<8, 8>(pl, sm.th, c, ew, inv, dfv, par); break;
              case 7: if (rows7) fast_plane<7, 7>(pl, sm.th, c, ew, inv, dfv, par); else fast_plane<7, 8>(pl, sm.th, c, ew, inv, dfv, par); break;
              case 6: if (rows7) fast_plane<6, 7>(pl, sm.th, c, ew, inv, dfv, par); else fast_plane<6, 8>(pl, sm.th, c, ew, inv, dfv, par); break;
              case 5: if (rows7) fast_plane<5, 7>(pl, sm.th, c, ew, inv, dfv, par); else fast_plane<5, 8>(pl, sm.th, c, ew, inv, dfv, par); break;
              default: if (rows7) fast_plane<4, 7>(pl, sm.th, c, ew, inv, dfv, par); else fast_plane<4, 8>(pl, sm.th, c, ew, inv, dfv, par); break;
            }
          } else
          switch (T.tv) {
            case 8: plain_plane<8>(pl, sm.th, sm.qd, c, T.tw, src, ew, inv, dn_fv, eout, S, par); break;
            case 7: plain_plane<7>(pl, sm.th, sm.qd, c, T.tw, src, ew, inv, dn_fv, eout, S, par); break;
            case 6: plain_plane<6>(pl, sm.th, sm.qd, c, T.tw, src, ew, inv, dn_fv, eout, S, par); break;
            case 5: plain_plane<5>(pl, sm.th, sm.qd, c, T.tw, src, ew, inv, dn_fv, eout, S, par); break;
            default: plain_plane<4>(pl, sm.th, sm.qd, c, T.tw, src, ew, inv, dn_fv, eout, S, par); break;
          }
          if (dn_fw) {  // the last row of the tile: still in ew unless the branch-free path computed rows beyond tw
            if ((src || eout) || T.tw == (rows7 ? 7 : 8)) {
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if (v < T.tv) dn_fw[v * kBrickRow] = tag(ew[v], par);
            } else {  // out of the plane buffer (the thread's own stores)
              const double *lrow = pl + (T.tw - 1) * kBrickTile * kP;
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if (v < T.tv) dn_fw[v * kBrickRow] = tag(lrow[v * kP], par);
            }
          }
        } else {
          // ---- per-cell path: holes and walls inside the tile (wall values straight from L2) ----------------------------------
          for (int w = 0; w < T.tw; ++w) {
            const unsigned long long frow = sm.flg[st][w];
            double ev = inv[0];
#pragma unroll
            for (int k = 0; k + 1 < kBrickTile; ++k) inv[k] = inv[k + 1];  // inv[0] is always the current row's v-face value
            if (frow == 0ull) continue;
            const int c0 = w * kBrickTile;
#pragma unroll 1
            for (int v = 0; v < T.tv; ++v) {
              const unsigned f = (unsigned)(frow >> (8 * v)) & 0xffu;
              double ewv = 0.0;
#pragma unroll
              for (int k = 0; k < kBrickTile; ++k) ewv = k == v ? ew[k] : ewv;
              if (f & BRK_ACT) {
                const int cell = c0 + v;
                double eu = pl[cell * kP];
                if (f & BRK_INJ_U) eu = __ldcg(irr + (int64_t)(ip++) * kBrickRow);
                if (f & BRK_INJ_V) ev = __ldcg(irr + (int64_t)(ip++) * kBrickRow);
                if (f & BRK_INJ_W) ewv = __ldcg(irr + (int64_t)(ip++) * kBrickRow);
                double r = c.k_th * sm.th[cell];
                if (f & BRK_SRC) r = fma(c.k_Q, sm.qd[cell], r);
                r = fma(c.c_w, ewv, fma(c.c_u, eu, r));
                const double e = fma(c.c_v, ev, r);
                pl[cell * kP] = e;
                ev = e;
                ewv = e;
                if (v + 1 == T.tv && dn_fv) dn_fv[w * kBrickRow] = tag(e, par);
                if (w + 1 == T.tw && dn_fw) dn_fw[v * kBrickRow] = tag(e, par);
                if (eout) __stcs(eout + cell * S, e);
              }
#pragma unroll
              for (int k = 0; k < kBrickTile; ++k) ew[k] = k == v ? ewv : ew[k];
            }
          }
        }
        if (dn_fv) dn_fv += kBrickTile * kBrickRow;
        if (dn_fw) dn_fw += kBrickTile * kBrickRow;
        if (eout) eout += kBrickCells * S;
      }
      PROF_T(p1);
      __syncthreads();  // B1: plane u is complete in the plane buffer; theta / Qdot of plane u are dead
      PROF_T(p2);
      bool early = false;
      if (!last_u) {
        stage(u + 1);
        // counter protocol only: the barrier orders every store of the CTA before this release (cumulativity)
        if (T.publish && t == 0) st_release(a.prog + task, (unsigned)(u + 1));
        // next plane's tile-face inflow: the loads fly during the reduction (counter faces: only if the upstream tile is
        // already there, otherwise after the reduction)
        early = !counters || ups.poll((unsigned)(u + 2));
        if (early) load_faces();
      }
      // ---- out of the plane buffer (thread = system): eps of the cells with an outgoing wall (closures), the u-face of the
      // segment ----------------------------------------------------------------------------------------------------------------
      if (on && T.wall_any) {
        for (int w = 0; w < T.tw; ++w) {
          const unsigned long long frow = sm.flg[st][w];
          if (frow & 0x2020202020202020ull) {
            const double *prow = sm.plane + w * kBrickTile * kP + s;
#pragma unroll
            for (int v = 0; v < kBrickTile; ++v)
              if ((frow >> (8 * v)) & BRK_WALL) {
                *wall = prow[v * kP];
                wall += kBrickRow;
              }
          }
        }
      }
      if (on && last_u && dn_fu) {
        for (int w = 0; w < T.tw; ++w) {
          const unsigned long long frow = sm.flg[st][w];
#pragma unroll
          for (int v = 0; v < kBrickTile; ++v)
            if ((frow >> (8 * v)) & BRK_ACT) dn_fu[(w * kBrickTile + v) * kBrickRow] = sm.plane[(w * kBrickTile + v) * kP + s];
        }
      }
      PROF_T(p3);
      // ------------------------------------------ moments: thread = one cell x half of the class's directions ------------------
      // a warp owns 16 cells (lanes 0-15 and 16-31 the two halves of the directions): one shuffle completes the sums, no
      // exchange between warps
      {
        const int mh = lane >> 4, cell = wid * 16 + (lane & 15);
        const int dh0 = (nd * mh) >> 1, dh1 = (nd * (mh + 1)) >> 1;
        const bool act = (reinterpret_cast<const unsigned char *>(sm.flg[st])[cell] & BRK_ACT) != 0;
        const double *mrow = sm.plane + cell * kP + dh0, *mdc = sm.dcoef + 4 * dh0;
        double m[5];
        switch (dh1 - dh0) {
          case 8: moments_cell<8>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 7: moments_cell<7>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 6: moments_cell<6>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 5: moments_cell<5>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 4: moments_cell<4>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 3: moments_cell<3>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 2: moments_cell<2>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          case 1: moments_cell<1>(mrow, sm.bcoef, mdc, G.nb, nd, m); break;
          default:
#pragma unroll
            for (int k = 0; k < 5; ++k) m[k] = 0.0;
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) m[k] += __shfl_xor_sync(0xffffffffu, m[k], 16);  // a + b on both sides: the same bits
        if (mh == 0 && act) {
          double *p = part + (int64_t)u * kBrickCells + cell;
#pragma unroll
          for (int k = 0; k < 5; ++k) p[k * npos] = m[k];
        }
        PROF_T(p4);
        if (!last_u) {
          if (!early) {
            ups.wait((unsigned)(u + 2));
            load_faces();
          }
          settle_faces();
        }
        PROF_T(p5);
        cp_async_wait_all();
        __syncthreads();  // B2: the plane buffer is free again; theta of plane u+1 has landed
        PROF_T(p6);
        PROF_ADD(0, p0, p1); PROF_ADD(1, p1, p2); PROF_ADD(2, p2, p3); PROF_ADD(3, p3, p4); PROF_ADD(4, p4, p5); PROF_ADD(5, p5, p6);
#ifdef BRICK_PROF
        if (t == 0) prof[6] += 1;
#endif
        if (last_u && t == 0) st_release(a.prog + task, 0x7fffffffu);
      }
    }
#ifdef BRICK_PROF
    if (t == 0) {
      for (int k = 0; k < 8; ++k) atomicAdd(&g_brick_prof[k], prof[k]);
      if (task < kBrickTlMax) {
        unsigned smid;
        asm volatile("mov.u32 %0, %smid;" : "=r"(smid));
        g_brick_tl[task][0] = tl0; g_brick_tl[task][1] = tl1; g_brick_tl[task][2] = gtime();
        g_brick_tl[task][3] = smid | ((unsigned long long)T.nu << 32) | ((unsigned long long)(T.tv * T.tw) << 48);
      }
    }
#endif
  }
}

}  // namespace

int nb_launch_sweep_brick(nanobte_solver *h, int store_e) {
  BrickState &bs = *h->brick;
  BrickArgs a = bs.a;
  a.store_e = store_e;
  bs.parity ^= 1u;
  a.parity = bs.parity;
  NB_CUDA(h, cudaMemsetAsync(a.ticket, 0, sizeof(unsigned int) * (size_t)(a.n_tasks + 1), h->stream));  // ticket + progress
  NB_CUDA(h, cudaFuncSetAttribute(sweep_brick_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BrickSmem)));
  sweep_brick_kernel<<<bs.grid, kBrickMaxS, sizeof(BrickSmem), h->stream>>>(a);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  bs.e_valid = store_e != 0;
  return 0;
}

size_t nb_brick_smem_bytes() { return sizeof(BrickSmem); }

#ifdef BRICK_PROF
extern "C" int nanobte_debug_brick_prof(unsigned long long *out, int reset) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(out, g_brick_prof, sizeof(unsigned long long) * 16);
  if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(g_brick_prof, z, sizeof(z)); }
  return 0;
}
extern "C" int nanobte_debug_brick_timeline(unsigned long long *out, int n_tasks) {  // [n_tasks][4] of the last sweep
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(out, g_brick_tl, sizeof(unsigned long long) * 4 * (size_t)std::min(n_tasks, kBrickTlMax));
  return 0;
}
#endif
