// kernels_brick.cu -- closures (a3), moment combine + temperature update (a6, a8) and exports for the row spaces of the
// tile-dataflow sweep (brick.h).  Same arithmetic as the kernels in kernels_common.cu, other addresses:
//   wall rows    eps of the cells with an outgoing boundary face, [row][system] per (class, group)
//   inflow rows  what the sweep reads at a wall (R6-R9), [row][system] per (class, group)
#include <algorithm>

#include "brick.h"

namespace {

__device__ __forceinline__ double nanmax_d(double a, double b) { return !(b <= a) ? b : a; }

struct BrickClosureArgs {
  BoundaryArgs a;
  double W;
  const BrickCG *cgs;
  const int32_t *cg_of;      // [n_cls][B]
  const int32_t *dir_local;  // [D]
  const int32_t *dir_cls;    // [D]
  const int32_t *cls_dirs;   // [n_cls][max_dirs]
  int32_t max_dirs;
  const double *wall;
  double *inf;
  // gsum
  const int32_t *out_bf[NB_MAX_CLASSES], *out_row[NB_MAX_CLASSES];
  const uint8_t *out_ord[NB_MAX_CLASSES];
  const BrickOutRow *out_rec[NB_MAX_CLASSES];
  int32_t n_out[NB_MAX_CLASSES];
  int32_t therm;             // 1: thermalizing faces only, 0: all the others
  double *partial;           // [4][n_bf][B]
  // inflow
  const int32_t *in_row[NB_MAX_CLASSES], *in_bf[NB_MAX_CLASSES];
  int32_t n_in[NB_MAX_CLASSES];
  int32_t n_rec[NB_MAX_CLASSES];
  const int32_t *bf_wrow;    // [n_cls][n_bf]
  int32_t init;
  // fast inflow kernel
  const BrickInRow *in_rec[NB_MAX_CLASSES];
  const uint8_t *in_perm;    // [n_cls][8][16]
  int32_t cg0[NB_MAX_CLASSES];
  int32_t n_cls;
};

// gnum share of one class: sum over the class's directions of w (s.n) eps at the wall cell (R7).  A warp walks over
// outgoing face entries of its class: per entry one 16-byte record (fetched one entry ahead), then the entry's wall rows (one
// per band group, S <= 128 contiguous doubles each) with coalesced loads, all in flight before the first use, through
// shared memory; lanes = bands then add the nd values of their band times w (s.n) in direction order (the arithmetic of a
// thread per (entry, band) walking its directions, bit for bit).
constexpr int kGsumGroups = 3;  // band groups covered by one pass (a class with more takes several)
constexpr int kGsumWarps = 4;
// A band's nd values sit at pitch nd + 1 (nd >= 8; fewer directions: no pad) and a group's block at pitch 146 (= 2 mod 16):
// with nd = 12 and 10 bands per group the 30 lanes of the summation hit 30 different banks in every half-warp.
constexpr int kGsumPitch = 146;
static_assert(kGsumPitch >= kBrickRow + kBrickRow / 8, "a row of 128 values with one pad per band of >= 8 directions");
__device__ __forceinline__ BrickOutRow ld_out_rec(const BrickOutRow *p) {
  const int4 r = __ldg(reinterpret_cast<const int4 *>(p));
  BrickOutRow o;
  o.bf = r.x; o.row = r.y; o.ord = (uint8_t)(r.z & 255); o.type = (uint8_t)((r.z >> 8) & 255);
  return o;
}
__global__ void __launch_bounds__(32 * kGsumWarps) brick_gsum_kernel(const BrickClosureArgs R) {
  __shared__ double buf[kGsumWarps][kGsumGroups * kGsumPitch];
  __shared__ double wsn[kGsumWarps][16];  // w (s.n) of the class's directions at the entry's face
  const BoundaryArgs &a = R.a;
  const int c = blockIdx.y, wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_out = R.n_out[c], stride = gridDim.x * kGsumWarps;
  int j = blockIdx.x * kGsumWarps + wid;
  if (j >= n_out) return;
  const int g0 = R.cg0[c], ng = R.cg_of[c * a.B + a.B - 1] - g0 + 1;
  const int nd = R.cgs[g0].nd, ndp = nd >= 8 ? nd + 1 : nd;
  double *mine = buf[wid];
  int S[kGsumGroups];
  int64_t wbase[kGsumGroups];
#pragma unroll
  for (int q = 0; q < kGsumGroups; ++q) {
    S[q] = q < ng ? R.cgs[g0 + q].S : 0;
    wbase[q] = q < ng ? R.cgs[g0 + q].wall_base : 0;
  }
  // lane = band (the bands beyond 32 and the groups beyond kGsumGroups take the general loops below)
  int my_q = -1, my_off = 0;
  double wd = 0.0;
  int dd = 0;
  if (lane < a.B) {
    my_q = R.cg_of[c * a.B + lane] - g0;
    my_off = my_q * kGsumPitch + (lane - R.cgs[g0 + my_q].b0) * ndp;
  }
  int pos[4];  // where value lane + 32 k of a row goes
#pragma unroll
  for (int k = 0; k < 4; ++k) pos[k] = lane + 32 * k + (ndp > nd ? (lane + 32 * k) / nd : 0);
  if (lane < nd) {
    dd = R.cls_dirs[c * R.max_dirs + lane];
    wd = a.w[dd];
  }
  BrickOutRow nxt = ld_out_rec(R.out_rec[c] + j);
  for (; j < n_out; j += stride) {
    const BrickOutRow rec = nxt;
    if (j + stride < n_out) nxt = ld_out_rec(R.out_rec[c] + j + stride);
    if ((rec.type == NANOBTE_THERMALIZING) != (R.therm != 0)) continue;
    double *out = R.partial + ((size_t)rec.ord * a.n_bf + rec.bf) * a.B;
    double v[kGsumGroups][4];
#pragma unroll
    for (int q = 0; q < kGsumGroups; ++q) {
      const double *src = R.wall + wbase[q] + (int64_t)rec.row * kBrickRow;
#pragma unroll
      for (int k = 0; k < 4; ++k) v[q][k] = lane + 32 * k < S[q] ? __ldg(src + lane + 32 * k) : 0.0;
    }
    if (lane < nd) wsn[wid][lane] = wd * a.bf_sn[(size_t)rec.bf * a.D + dd];
#pragma unroll
    for (int q = 0; q < kGsumGroups; ++q) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (lane + 32 * k < S[q]) mine[q * kGsumPitch + pos[k]] = v[q][k];
    }
    __syncwarp();
    if (my_q >= 0 && my_q < kGsumGroups) {
      double acc = 0.0;
      for (int dl = 0; dl < nd; ++dl) acc = fma(wsn[wid][dl], mine[my_off + dl], acc);
      out[lane] = acc;
    }
    for (int b = lane + 32; b < a.B; b += 32) {  // more than 32 bands
      const int q = R.cg_of[c * a.B + b] - g0;
      if (q >= kGsumGroups) continue;
      const int off = q * kGsumPitch + (b - R.cgs[g0 + q].b0) * ndp;
      double acc = 0.0;
      for (int dl = 0; dl < nd; ++dl) acc = fma(wsn[wid][dl], mine[off + dl], acc);
      out[b] = acc;
    }
    for (int gb = kGsumGroups; gb < ng; ++gb) {  // more than kGsumGroups band groups: one group at a time
      __syncwarp();
      const BrickCG &G = R.cgs[g0 + gb];
      const double *src = R.wall + G.wall_base + (int64_t)rec.row * kBrickRow;
      for (int e = lane; e < G.S; e += 32) mine[e] = __ldg(src + e);
      __syncwarp();
      for (int bl = lane; bl < G.nb; bl += 32) {
        double acc = 0.0;
        for (int dl = 0; dl < nd; ++dl) acc = fma(wsn[wid][dl], mine[bl * nd + dl], acc);
        out[G.b0 + bl] = acc;
      }
    }
    __syncwarp();
  }
}

// Inflow rows of the boundary faces (R6-R8, lagged R9): one CTA per (row, (class, group)), lanes = systems.
__global__ void __launch_bounds__(kBrickMaxS) brick_inflow_kernel(const BrickClosureArgs R) {
  const BoundaryArgs &a = R.a;
  const BrickCG G = R.cgs[blockIdx.y];
  const int c = G.cls, k = blockIdx.x, s = threadIdx.x;
  if (k >= R.n_in[c] || s >= G.S) return;
  const int bf = R.in_bf[c][k];
  const int type = a.bf_type[bf];
  double *dst = R.inf + G.inf_base + (int64_t)R.in_row[c][k] * kBrickRow + s;
  const int b = G.b0 + s / G.nd;
  if (type == NANOBTE_THERMALIZING) {
    if (R.init) *dst = a.C[b] * a.bf_eps_w[bf] / R.W;  // R6; never changes afterwards
    return;
  }
  if (R.init) return;  // eps^0 = 0 (R12)
  const double Gf = a.G[(size_t)bf * a.B + b];
  if (type == NANOBTE_DIFFUSE) {
    *dst = Gf;  // R7
    return;
  }
  const int d = R.cls_dirs[c * R.max_dirs + s % G.nd];
  const int md = a.bf_mirror[(size_t)bf * a.D + d];
  if (md < 0) {  // s_d . n == 0 exactly (R15): the sweep multiplies this row by 0
    *dst = 0.0;
    return;
  }
  const int cm = R.dir_cls[md];
  const BrickCG Gm = R.cgs[R.cg_of[cm * a.B + b]];
  const double spec = R.wall[Gm.wall_base + (int64_t)R.bf_wrow[(size_t)cm * a.n_bf + bf] * kBrickRow + (b - Gm.b0) * Gm.nd + R.dir_local[md]];
  *dst = type == NANOBTE_SPECULAR ? spec : a.bf_p[bf] * spec + (1.0 - a.bf_p[bf]) * Gf;  // R8
}

// The same from the per-row records built at create (BrickInRow), for every launch but the first (R.init, general kernel):
// a CTA belongs to one (class, group), lanes = systems, and walks over the class's records kBrickInRows at a time; the
// records are sorted by face type and padded, so a batch has one type and takes one uniform branch into straight-line code.
// What does not depend on the row is set up once per CTA: the thread's band and direction, its mirror direction under each
// of the class's (at most 8) permutations packed in one register, the wall block of this band group in every class (the
// classes have the same directions per band here, BrickState::in_fast).  Per row: one 16-byte record (uniform; the next
// batch's records are fetched while these are worked on), then G / p / the wall value (independent loads), then
//   diffuse G (R7)    specular: the mirror value    mixed: p spec + (1 - p) G (R8)    0 where s.n == 0 (R15).
constexpr int kInRows = kBrickInRows;
__global__ void __launch_bounds__(kBrickMaxS) brick_inflow_fast_kernel(const BrickClosureArgs R) {
  __shared__ int64_t m_base[NB_MAX_CLASSES];
  const BoundaryArgs &a = R.a;
  const BrickCG G = R.cgs[blockIdx.y];
  const int c = G.cls, s = threadIdx.x;
  const int g = blockIdx.y - R.cg0[c];           // band group index: the same in the mirror class
  if (s < R.n_cls) m_base[s] = R.cgs[R.cg0[s] + g].wall_base;
  __syncthreads();
  const int n_rec = R.n_rec[c];
  if (s >= G.S) return;
  const int bl = s / G.nd, dl = s - bl * G.nd;
  unsigned long long perms = 0;                  // byte q: mirror direction (local to its class) under permutation q, 255 = none
#pragma unroll
  for (int q = 0; q < 8; ++q) perms |= (unsigned long long)R.in_perm[((size_t)c * 8 + q) * 16 + dl] << (8 * q);
  double *inf = R.inf + G.inf_base + s;
  const double *Gb = a.G + G.b0 + bl;
  const double *wall = R.wall + bl * G.nd;
  const int4 *recs = reinterpret_cast<const int4 *>(R.in_rec[c]);
  const int stride = gridDim.x * kInRows;
  int4 nxt[kInRows];  // x: face (-1: padding), y: inflow row, z: wall row of the mirror cell, w: type | mirror class << 8 | permutation << 16
  if (blockIdx.x * kInRows < n_rec) {
#pragma unroll
    for (int q = 0; q < kInRows; ++q) nxt[q] = __ldg(recs + blockIdx.x * kInRows + q);
  }
  for (int k0 = blockIdx.x * kInRows; k0 < n_rec; k0 += stride) {
    int4 rec[kInRows];
#pragma unroll
    for (int q = 0; q < kInRows; ++q) rec[q] = nxt[q];
    if (k0 + stride < n_rec) {
#pragma unroll
      for (int q = 0; q < kInRows; ++q) nxt[q] = __ldg(recs + k0 + stride + q);
    }
    const int type = rec[0].w & 255;
    if (type == NANOBTE_DIFFUSE) {
      double Gf[kInRows];
#pragma unroll
      for (int q = 0; q < kInRows; ++q) Gf[q] = rec[q].x >= 0 ? Gb[(size_t)rec[q].x * a.B] : 0.0;
#pragma unroll
      for (int q = 0; q < kInRows; ++q)
        if (rec[q].x >= 0) inf[(int64_t)rec[q].y * kBrickRow] = Gf[q];
      continue;
    }
    bool mir[kInRows];
    double spec[kInRows];
#pragma unroll
    for (int q = 0; q < kInRows; ++q) {
      const int cm = (rec[q].w >> 8) & 255, perm = (rec[q].w >> 16) & 255;
      const int dlm = (int)((perms >> (8 * perm)) & 255ull);
      mir[q] = rec[q].x >= 0 && rec[q].z >= 0 && dlm != 255;
      spec[q] = mir[q] ? wall[m_base[cm] + (int64_t)rec[q].z * kBrickRow + dlm] : 0.0;
    }
    if (type == NANOBTE_SPECULAR) {
#pragma unroll
      for (int q = 0; q < kInRows; ++q)
        if (rec[q].x >= 0) inf[(int64_t)rec[q].y * kBrickRow] = spec[q];
      continue;
    }
    double Gf[kInRows], p[kInRows];
#pragma unroll
    for (int q = 0; q < kInRows; ++q) {
      Gf[q] = mir[q] ? Gb[(size_t)rec[q].x * a.B] : 0.0;
      p[q] = rec[q].x >= 0 ? a.bf_p[rec[q].x] : 0.0;
    }
#pragma unroll
    for (int q = 0; q < kInRows; ++q)
      if (rec[q].x >= 0) inf[(int64_t)rec[q].y * kBrickRow] = mir[q] ? p[q] * spec[q] + (1.0 - p[q]) * Gf[q] : 0.0;
  }
}

// Combine the partials of every (class, group) per cell in fixed order, update T, track max |dT|, refresh the
// sweep-order copies of theta.
struct BrickUpdateArgs {
  int32_t n_act, n_cls, n_cg, mode;
  const BrickCG *cgs;
  const double *part;
  int32_t npos[NB_MAX_CLASSES];
  const int32_t *a2pos;  // [n_cls][n_act]
  const int32_t *pos2a;  // [npos[0]] cell at a position of class 0 (-1: none): threads follow the positions, so that the loads of
                         // the partial moments are coalesced (the tiles are the same lattice in every class)
  double *th[NB_MAX_CLASSES];
  double *theta, *theta_prev, *theta_SI, *theta_en, *q;
  const double *x;
  double beta, Csum;
  unsigned long long *maxdT;
};

__global__ void __launch_bounds__(256) brick_update_kernel(const BrickUpdateArgs u) {
  __shared__ double red[8];
  const int p0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int a = p0 < u.npos[0] ? u.pos2a[p0] : -1;
  double d = 0.0;
  if (a >= 0) {
    double th;
    if (u.mode == 0) {
      double m[5] = {0, 0, 0, 0, 0};
      for (int g = 0; g < u.n_cg; ++g) {
        const int c = u.cgs[g].cls;
        const double *p = u.part + u.cgs[g].part_base + u.a2pos[(size_t)c * u.n_act + a];
#pragma unroll
        for (int k = 0; k < 5; ++k) m[k] += p[(size_t)k * u.npos[c]];
      }
      th = m[0] / u.beta;               // Eq. 5
      u.theta_SI[a] = th;
      u.theta_en[a] = m[1] / u.Csum;    // R13
      u.q[3 * (size_t)a] = m[2];        // Eq. 7
      u.q[3 * (size_t)a + 1] = m[3];
      u.q[3 * (size_t)a + 2] = m[4];
      u.theta_prev[a] = u.theta[a];
    } else {
      th = u.theta_SI[a] + u.x[a];      // R14a
    }
    u.theta[a] = th;                    // Eq. 6
    d = fabs(th - u.theta_prev[a]);
    for (int c = 0; c < u.n_cls; ++c) u.th[c][u.a2pos[(size_t)c * u.n_act + a]] = th;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) d = nanmax_d(d, __shfl_xor_sync(0xffffffffu, d, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = d;
  __syncthreads();
  if (threadIdx.x < 32) {
    d = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d = nanmax_d(d, __shfl_xor_sync(0xffffffffu, d, o));
    if (threadIdx.x == 0) atomicMax(u.maxdT, (unsigned long long)__double_as_longlong(d));
  }
}

__global__ void brick_set_theta_kernel(int n_act, int n_cls, const int32_t *act2cell, const double *T, double T_ref,
                                       double *theta, const int32_t *a2pos, BrickUpdateArgs u) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_act) return;
  const double th = T[act2cell[a]] - T_ref;
  theta[a] = th;
  for (int c = 0; c < n_cls; ++c) u.th[c][a2pos[(size_t)c * n_act + a]] = th;
}

struct BrickGetEArgs {
  int32_t n_cells, n_act, B, b0, nb, d0, nd;
  const int32_t *cell2act, *a2pos, *dir_cls, *dir_local, *cg_of;
  const BrickCG *cgs;
  const double *e, *C;
  double off_scale;
  double *dst;
};

__global__ void brick_get_e_kernel(const BrickGetEArgs g) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.n_cells) return;
  const int bi = blockIdx.y / g.nd, di = blockIdx.y % g.nd;
  const int b = g.b0 + bi, d = g.d0 + di;
  const int a = g.cell2act[c];
  double val = 0.0;
  if (a >= 0) {
    const int cls = g.dir_cls[d];
    const BrickCG G = g.cgs[g.cg_of[cls * g.B + b]];
    const int64_t pos = g.a2pos[(size_t)cls * g.n_act + a];
    val = g.e[G.e_base + pos * G.S + (b - G.b0) * G.nd + g.dir_local[d]] + g.C[b] * g.off_scale;
  }
  g.dst[((size_t)bi * g.nd + di) * g.n_cells + c] = val;
}

BrickClosureArgs closure_args(nanobte_solver *h) {
  const BrickState &bs = *h->brick;
  BrickClosureArgs R{};
  R.a = h->bd; R.W = h->W; R.cgs = bs.a.cgs; R.cg_of = bs.cg_of; R.dir_local = bs.dir_local; R.dir_cls = h->dir_cls;
  R.cls_dirs = h->cls_dirs; R.max_dirs = h->max_cls_dirs; R.wall = bs.a.wall; R.inf = bs.a.inf; R.partial = h->g_partial;
  R.bf_wrow = bs.bf_wrow;
  R.in_perm = bs.in_perm;
  R.n_cls = h->n_cls;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) {
    R.in_rec[c] = bs.in_rec[c]; R.cg0[c] = bs.cg0[c];
    R.out_bf[c] = bs.out_bf[c]; R.out_row[c] = bs.out_row[c]; R.out_ord[c] = bs.out_ord[c]; R.n_out[c] = bs.n_out[c];
    R.out_rec[c] = bs.out_rec[c];
    R.in_row[c] = bs.in_row[c]; R.in_bf[c] = bs.in_bf[c]; R.n_in[c] = bs.n_in[c]; R.n_rec[c] = bs.n_rec[c];
  }
  return R;
}

int launch_gsum(nanobte_solver *h, const int32_t *faces, int n_faces, int therm) {
  if (n_faces == 0) return 0;
  BrickClosureArgs R = closure_args(h);
  R.therm = therm;
  int64_t nmax = 0;
  for (int c = 0; c < h->n_cls; ++c) nmax = std::max<int64_t>(nmax, R.n_out[c]);
  if (nmax > 0) {
    // a few waves of CTAs; each warp walks over its share of the entries
    const int64_t want = ((int64_t)32 * h->n_sm + h->n_cls - 1) / h->n_cls;
    dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>((nmax + kGsumWarps - 1) / kGsumWarps, want)), h->n_cls);
    brick_gsum_kernel<<<grid, 128, 0, h->stream>>>(R);
    h->launches++;
    NB_CUDA(h, cudaGetLastError());
  }
  return nb_launch_gcomb(h, faces, n_faces, h->brick->bf_nord);
}

int launch_inflow(nanobte_solver *h, int init) {
  BrickClosureArgs R = closure_args(h);
  R.init = init;
  int nmax = 0;
  for (int c = 0; c < h->n_cls; ++c) nmax = std::max(nmax, R.n_in[c]);
  if (nmax == 0) return 0;
  if (h->brick->in_fast && !init) {
    int rmax = 0;
    for (int c = 0; c < h->n_cls; ++c) rmax = std::max(rmax, R.n_rec[c]);
    if (rmax == 0) return 0;  // thermalizing faces only: nothing changes after the first launch
    // a few waves of CTAs; each walks over its share of the records
    const int want = (32 * h->n_sm + h->brick->n_cg - 1) / h->brick->n_cg;
    dim3 grid(std::max(1, std::min(rmax / kInRows, want)), h->brick->n_cg);
    brick_inflow_fast_kernel<<<grid, kBrickMaxS, 0, h->stream>>>(R);
  } else {
    dim3 grid(nmax, h->brick->n_cg);
    brick_inflow_kernel<<<grid, kBrickMaxS, 0, h->stream>>>(R);
  }
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

BrickUpdateArgs update_args(nanobte_solver *h, int mode) {
  const BrickState &bs = *h->brick;
  BrickUpdateArgs u{};
  u.n_act = h->n_act; u.n_cls = h->n_cls; u.n_cg = bs.n_cg; u.mode = mode; u.cgs = bs.a.cgs; u.part = bs.a.part;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) { u.npos[c] = bs.a.npos[c]; u.th[c] = bs.th[c]; }
  u.a2pos = bs.a2pos;
  u.pos2a = bs.pos2a;
  u.theta = h->theta; u.theta_prev = h->theta_prev; u.theta_SI = h->theta_SI; u.theta_en = h->theta_en; u.q = h->q;
  u.x = h->cg_x; u.beta = h->beta; u.Csum = h->Csum; u.maxdT = h->d_maxdT;
  return u;
}

}  // namespace

int nb_brick_closures(nanobte_solver *h, int init) {
  if (h->n_bf == 0) return 0;
  h->therm_stale = true;
  if (init) return launch_inflow(h, 1);
  if (h->n_refl == 0) return 0;
  int rc = launch_gsum(h, h->refl_faces, h->n_refl, 0);
  if (rc < 0) return rc;
  return launch_inflow(h, 0);
}

int nb_brick_refresh_thermalizing(nanobte_solver *h) {
  if (!h->therm_stale) return 0;
  int rc = launch_gsum(h, h->therm_faces, h->n_therm, 1);
  if (rc < 0) return rc;
  h->therm_stale = false;
  return 0;
}

int nb_brick_update(nanobte_solver *h, int mode) {
  BrickUpdateArgs u = update_args(h, mode);
  brick_update_kernel<<<(u.npos[0] + 255) / 256, 256, 0, h->stream>>>(u);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

int nb_brick_set_theta(nanobte_solver *h, const double *T_cells_dev) {
  BrickUpdateArgs u = update_args(h, 0);
  brick_set_theta_kernel<<<(h->n_act + 255) / 256, 256, 0, h->stream>>>(h->n_act, h->n_cls, h->act2cell, T_cells_dev, h->T_ref,
                                                                         h->theta, h->brick->a2pos, u);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

int nb_brick_get_e(nanobte_solver *h, int b0, int nb, int d0, int nd, double *dst_dev, int deviational) {
  if (nb == 0 || nd == 0) return 0;
  const BrickState &bs = *h->brick;
  BrickGetEArgs g{};
  g.n_cells = h->n_cells; g.n_act = h->n_act; g.B = h->B; g.b0 = b0; g.nb = nb; g.d0 = d0; g.nd = nd;
  g.cell2act = h->cell2act; g.a2pos = bs.a2pos; g.dir_cls = h->dir_cls; g.dir_local = bs.dir_local; g.cg_of = bs.cg_of;
  g.cgs = bs.a.cgs; g.e = bs.a.e; g.C = h->bd.C; g.off_scale = deviational ? 0.0 : h->T_ref / h->W; g.dst = dst_dev;
  dim3 grid((h->n_cells + 255) / 256, nb * nd);
  brick_get_e_kernel<<<grid, 256, 0, h->stream>>>(g);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

void nb_free_brick(nanobte_solver *h) {
  delete h->brick;
  h->brick = nullptr;
}
