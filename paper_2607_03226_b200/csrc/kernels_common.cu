// kernels_common.cu -- kernels shared by both mesh kinds: boundary closures (a3), moment reduction (a6),
// temperature update (a8), exports, and the conjugate-gradient diffusion correction (a7).
// Everything is fp64, deterministic (no floating-point atomics; fixed reduction trees).
#include <cooperative_groups.h>

#include <algorithm>

#include "brick.h"
namespace cg = cooperative_groups;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double nanmax(double a, double b) { return !(b <= a) ? b : a; }  // NaN wins
__device__ __forceinline__ double warp_nanmax(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// =================================================================================================================
// (a3) boundary closures, one warp per boundary face, lanes over directions, loop over bands.
//   G_bf   = sum_{s.n>0} w (s.n) eps_{b,s,c} / sum_{s.n<0} w |s.n|                     (R7)
//   inflow = thermalizing C_b (T_w - T_ref)/W (R6) | G (diffuse) | eps_{b,r(s),c} (specular) | p spec + (1-p) G (R8)
//   faceflux_bf,b = v_b [ sum_out w (s.n) eps^{n+1} + sum_in w (s.n) inflow^{n} ]       (O8; inflow^n = what the
//                   sweep that produced eps^{n+1} consumed -- read before it is overwritten)
// =================================================================================================================
struct BoundaryRun {
  BoundaryArgs a;
  double W;
  int unstructured;  // e layout [D][n_pos][B] instead of [D][B][n_pos]
};

__global__ void __launch_bounds__(256) boundary_kernel(BoundaryRun R) {
  extern __shared__ double sm[];
  const BoundaryArgs &a = R.a;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int bf = blockIdx.x * (blockDim.x >> 5) + wib;
  if (bf >= a.n_bf) return;
  double *eo = sm + (size_t)wib * a.D;
  const int type = a.bf_type[bf];
  const double p = a.bf_p[bf], den = a.bf_den[bf], dTw = a.bf_eps_w[bf];
  const size_t row = (size_t)bf * a.D;
  for (int b = 0; b < a.B; ++b) {
    double gnum = 0.0;
    for (int d = lane; d < a.D; d += 32) {
      const double sn = a.bf_sn[row + d];
      if (sn > 0.0) {
        const int64_t pos = a.bf_opos[row + d];
        const double val = R.unstructured ? a.e[((int64_t)d * a.e_stride + pos) * a.B + b]
                                          : a.e[((int64_t)a.dir_row0[d] + b) * a.e_stride + pos];
        eo[d] = val;
        gnum += a.w[d] * sn * val;
      }
    }
    gnum = warp_sum(gnum);
    __syncwarp();
    const double Gb = den > 0.0 ? gnum / den : 0.0;
    double fin = 0.0;
    for (int d = lane; d < a.D; d += 32) {
      const double sn = a.bf_sn[row + d];
      if (sn < 0.0) {
        const int64_t addr = a.dir_bin[d] + (int64_t)b * a.dir_nin[d] + a.bf_inidx[row + d];
        fin += a.w[d] * sn * a.bin[addr];
        double nv;
        if (type == NANOBTE_THERMALIZING) nv = a.C[b] * dTw / R.W;
        else if (type == NANOBTE_DIFFUSE) nv = Gb;
        else {
          const double spec = eo[a.bf_mirror[row + d]];
          nv = (type == NANOBTE_SPECULAR) ? spec : p * spec + (1.0 - p) * Gb;
        }
        a.bin[addr] = nv;
      }
    }
    fin = warp_sum(fin);
    if (lane == 0) {
      a.G[(size_t)bf * a.B + b] = Gb;
      a.faceflux[(size_t)bf * a.B + b] = a.v[b] * (gnum + fin);
    }
    __syncwarp();
  }
}

static int launch_closure_G(nanobte_solver *h, const int32_t *faces, int n_faces, int therm);
static int launch_closure_inflow(nanobte_solver *h, int init);

int nb_launch_boundary(nanobte_solver *h, int init) {
  if (h->n_bf == 0) return 0;
  if (h->brick) return nb_brick_closures(h, init);
  if (h->split_closures) {
    h->therm_stale = true;
    if (init) return launch_closure_inflow(h, 1);
    if (h->n_refl == 0) return 0;
    int rc = launch_closure_G(h, h->refl_faces, h->n_refl, 0);
    if (rc < 0) return rc;
    return launch_closure_inflow(h, 0);
  }
  BoundaryRun R;
  R.a = h->bd;
  R.W = h->W;
  R.unstructured = h->kind;
  const int wpb = 8;
  const size_t smem = (size_t)wpb * h->D * sizeof(double);
  boundary_kernel<<<(h->n_bf + wpb - 1) / wpb, wpb * 32, smem, h->stream>>>(R);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// =================================================================================================================
// (a3) structured grids: the closures as two kernels whose global accesses follow the memory layout.
//   closure_gsum_kernel   one thread per (octant class, wall cell that is outgoing for the class, chunk of bands): the
//                         class's share of gnum = sum_out w (s.n) eps.  Lanes run over wall cells in position
//                         order, which are contiguous in every e row (a hyperplane stores its wall cells first).
//   closure_gcomb_kernel  G_bf (R7) from the class partials in fixed order, and the face flux (O8).  The incoming
//                         half of the flux needs no gather: the inflow the last sweep consumed was C_b dT_w/W
//                         (thermalizing) or built from
//                         eps^{n-1} with G^{n-1}, and sum_in w (s.n) inflow = -den * G^{n-1} for diffuse, specular and
//                         mixed walls alike because the quadrature is mirror symmetric about the wall (weights
//                         checked at create), so  F_bf = v_b (gnum^n - den * X),  X = C_b dT_w/W  or  G^{n-1}_bf.
//   closure_inflow_kernel one thread per (octant class, slot of its inflow row, direction of the class): writes the
//                         inflow cache in exactly the order the sweep's bulk loads read it -> coalesced stores;
//                         the specular part gathers eps of the mirrored direction (R8).
// Thermalizing faces never change their inflow (written once at create) and their G / flux are diagnostics only:
// they are skipped per iteration and evaluated on demand (get_G, get_boundary_heat).
// =================================================================================================================
struct GsumArgs {
  BoundaryArgs a;
  const int32_t *out_bf[NB_MAX_CLASSES];   // per class: boundary faces that are OUTGOING for the class, in position order
  const int32_t *out_pos[NB_MAX_CLASSES];  //            position of the wall cell in the class's e rows
  const uint8_t *out_ord[NB_MAX_CLASSES];  //            which of the face's outgoing classes this is (0..3)
  int32_t cls_nout[NB_MAX_CLASSES], cls_ndirs[NB_MAX_CLASSES];
  const int32_t *cls_dirs;                 // [n_cls][max_dirs]
  int32_t max_dirs, bands_per_chunk, therm;  // therm: 1 = thermalizing faces only, 0 = all the others
  double *partial;                         // [4][n_bf][B]
};

// gnum partials: sum over the directions of ONE class of w (s.n) eps at the wall cell.  Lanes run over the wall cells
// of a class in position order -- contiguous in every e row because a hyperplane stores its wall cells first.
constexpr int kGsumUB = 6;
__global__ void __launch_bounds__(128) closure_gsum_kernel(GsumArgs R) {
  const BoundaryArgs &a = R.a;
  const int c = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= R.cls_nout[c]) return;
  const int bf = R.out_bf[c][j];
  if ((a.bf_type[bf] == NANOBTE_THERMALIZING) != (R.therm != 0)) return;
  const int b_lo = blockIdx.z * R.bands_per_chunk;
  const int nb = min(a.B - b_lo, R.bands_per_chunk);
  const double *src0 = a.e + R.out_pos[c][j] + (int64_t)b_lo * a.e_stride;
  const double *sn = a.bf_sn + (size_t)bf * a.D;
  for (int b0 = 0; b0 < nb; b0 += kGsumUB) {
    double acc[kGsumUB];
#pragma unroll
    for (int u = 0; u < kGsumUB; ++u) acc[u] = 0.0;
    for (int kd = 0; kd < R.cls_ndirs[c]; ++kd) {
      const int d = R.cls_dirs[c * R.max_dirs + kd];
      const double wsn = a.w[d] * sn[d];
      const double *src = src0 + ((int64_t)a.dir_row0[d] + b0) * a.e_stride;
      double v[kGsumUB];
#pragma unroll
      for (int u = 0; u < kGsumUB; ++u) v[u] = __ldcs(src + (int64_t)min(u, nb - 1 - b0) * a.e_stride);
#pragma unroll
      for (int u = 0; u < kGsumUB; ++u) acc[u] += wsn * v[u];
    }
    double *dst = R.partial + ((size_t)R.out_ord[c][j] * a.n_bf + bf) * a.B + b_lo + b0;
#pragma unroll
    for (int u = 0; u < kGsumUB; ++u)
      if (b0 + u < nb) dst[u] = acc[u];
  }
}

struct GcombArgs {
  BoundaryArgs a;
  double W;
  const int32_t *faces;      // face list this launch covers
  const uint8_t *nord;       // [n_bf] number of outgoing classes of the face
  const double *partial;
  int32_t n_faces;
};

// G_bf = (sum of the class partials, fixed order) / den (R7); face flux (O8) with the lagged inflow in closed form.
__global__ void __launch_bounds__(256) closure_gcomb_kernel(GcombArgs R) {
  const BoundaryArgs &a = R.a;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)R.n_faces * a.B) return;
  const int bf = R.faces[i / a.B], b = (int)(i % a.B);
  double gnum = 0.0;
  for (int o = 0; o < R.nord[bf]; ++o) gnum += R.partial[((size_t)o * a.n_bf + bf) * a.B + b];
  const double den = a.bf_den[bf];
  const size_t k = (size_t)bf * a.B + b;
  const double Gold = a.G[k];
  a.G[k] = den > 0.0 ? gnum / den : 0.0;
  const double X = a.bf_type[bf] == NANOBTE_THERMALIZING ? a.C[b] * a.bf_eps_w[bf] / R.W : Gold;
  a.faceflux[k] = a.v[b] * (gnum - den * X);
}

struct InflowArgs {
  BoundaryArgs a;
  double W;
  const int32_t *cls_inbf[NB_MAX_CLASSES];  // per class: face id of every slot of the inflow row (-1 = padding)
  int32_t cls_nin[NB_MAX_CLASSES], cls_ndirs[NB_MAX_CLASSES];
  const int32_t *cls_dirs;                   // [n_cls][max_dirs]
  int32_t max_dirs, init;
};

__global__ void __launch_bounds__(128) closure_inflow_kernel(InflowArgs R) {
  const BoundaryArgs &a = R.a;
  const int c = blockIdx.y, kd = blockIdx.z;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (kd >= R.cls_ndirs[c] || idx >= R.cls_nin[c]) return;
  const int bf = R.cls_inbf[c][idx];
  if (bf < 0) return;
  const int type = a.bf_type[bf];
  const int d = R.cls_dirs[c * R.max_dirs + kd];
  const int64_t n_in = a.dir_nin[d];
  double *dst = a.bin + a.dir_bin[d] + idx;
  if (type == NANOBTE_THERMALIZING) {
    if (R.init) {
      const double dTw = a.bf_eps_w[bf];
      for (int b = 0; b < a.B; ++b) dst[b * n_in] = a.C[b] * dTw / R.W;  // R6
    }
    return;
  }
  if (R.init) return;  // eps^0 = 0 (R12): reflecting walls start from a zero cache
  const double *Gf = a.G + (size_t)bf * a.B;
  if (type == NANOBTE_DIFFUSE) {
    for (int b = 0; b < a.B; ++b) dst[b * n_in] = Gf[b];  // R7
    return;
  }
  const double p = type == NANOBTE_SPECULAR ? 1.0 : a.bf_p[bf];
  const int md = a.bf_mirror[(size_t)bf * a.D + d];
  if (md < 0) {  // s_d . n == 0 exactly (R15): the face carries nothing for d; the sweep multiplies this slot by |s.n|/h = 0
    for (int b = 0; b < a.B; ++b) dst[b * n_in] = 0.0;
    return;
  }
  const double *src = a.e + (int64_t)a.dir_row0[md] * a.e_stride + a.bf_opos[(size_t)bf * a.D + md];
  constexpr int UB = 6;
  for (int b0 = 0; b0 < a.B; b0 += UB) {
    double spec[UB];
#pragma unroll
    for (int j = 0; j < UB; ++j) spec[j] = __ldcs(src + (int64_t)min(b0 + j, a.B - 1) * a.e_stride);
#pragma unroll
    for (int j = 0; j < UB; ++j)
      if (b0 + j < a.B) dst[(b0 + j) * n_in] = type == NANOBTE_SPECULAR ? spec[j] : p * spec[j] + (1.0 - p) * Gf[b0 + j];  // R8
  }
}

static int launch_closure_G(nanobte_solver *h, const int32_t *faces, int n_faces, int therm) {
  if (n_faces == 0) return 0;
  GsumArgs S;
  S.a = h->bd; S.cls_dirs = h->cls_dirs; S.max_dirs = h->max_cls_dirs; S.therm = therm; S.partial = h->g_partial;
  int nout_max = 0;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) {
    S.out_bf[c] = h->cls_outbf[c]; S.out_pos[c] = h->cls_outpos[c]; S.out_ord[c] = h->cls_outord[c];
    S.cls_nout[c] = h->cls_nout[c]; S.cls_ndirs[c] = h->cls_ndirs[c];
    nout_max = std::max(nout_max, h->cls_nout[c]);
  }
  S.bands_per_chunk = kGsumUB;
  dim3 grid((nout_max + 127) / 128, h->n_cls, (h->B + kGsumUB - 1) / kGsumUB);
  closure_gsum_kernel<<<grid, 128, 0, h->stream>>>(S);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return nb_launch_gcomb(h, faces, n_faces, h->bf_nord);
}

// G_bf and the face flux of the listed faces from the per-class shares in g_partial (nord[f] shares of face f).
int nb_launch_gcomb(nanobte_solver *h, const int32_t *faces, int n_faces, const uint8_t *nord) {
  if (n_faces == 0) return 0;
  GcombArgs R;
  R.a = h->bd; R.W = h->W; R.faces = faces; R.nord = nord; R.partial = h->g_partial; R.n_faces = n_faces;
  const int64_t n = (int64_t)n_faces * h->B;
  closure_gcomb_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(R);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

static int launch_closure_inflow(nanobte_solver *h, int init) {
  InflowArgs R;
  R.a = h->bd; R.W = h->W; R.cls_dirs = h->cls_dirs; R.max_dirs = h->max_cls_dirs; R.init = init;
  int nin_max = 0;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) {
    R.cls_inbf[c] = h->cls_inbf[c];
    R.cls_nin[c] = h->cls_nin[c];
    R.cls_ndirs[c] = h->cls_ndirs[c];
    nin_max = std::max(nin_max, h->cls_nin[c]);
  }
  if (nin_max == 0) return 0;
  dim3 grid((nin_max + 127) / 128, h->n_cls, h->max_cls_dirs);
  closure_inflow_kernel<<<grid, 128, 0, h->stream>>>(R);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// Diagnostics of the thermalizing faces (G, face flux) from the current eps; called by the getters that expose them.
int nb_refresh_thermalizing(nanobte_solver *h) {
  if (h->brick) return nb_brick_refresh_thermalizing(h);
  if (!h->split_closures || !h->therm_stale) return 0;
  int rc = launch_closure_G(h, h->therm_faces, h->n_therm, 1);
  if (rc < 0) return rc;
  h->therm_stale = false;
  return 0;
}

// =================================================================================================================
// (a6) moments, structured layout.  One thread per pair of positions of one class (octant); streams every e row
// of the class exactly once (8 B per update) and writes the class's partial sums
//   part[c][0] = sum w/tau eps   part[c][1] = sum w eps   part[c][2..4] = sum v w s eps      (Eq. 5, R13, Eq. 7)
// =================================================================================================================
struct MomentsArgs {
  const double *e;
  const double *mcoef;  // [rows][5]
  double *part;
  int64_t e_stride;
  int32_t cls_nsys[NB_MAX_CLASSES], cls_row0[NB_MAX_CLASSES], cls_npos[NB_MAX_CLASSES];
};

__global__ void __launch_bounds__(256) moments_structured_kernel(MomentsArgs a) {
  extern __shared__ double smc[];  // [nsys][5]
  const int c = blockIdx.y;
  const int nsys = a.cls_nsys[c];
  const int64_t row0 = a.cls_row0[c];
  for (int k = threadIdx.x; k < nsys * 5; k += blockDim.x) smc[k] = a.mcoef[(size_t)row0 * 5 + k];
  __syncthreads();
  const int64_t pos = 2 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (pos >= a.cls_npos[c]) return;
  double2 m0 = {0, 0}, m1 = {0, 0}, m2 = {0, 0}, m3 = {0, 0}, m4 = {0, 0};
  const double *base = a.e + row0 * a.e_stride + pos;
  int k = 0;
  for (; k + 4 <= nsys; k += 4) {
    double2 v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) v[j] = __ldcs(reinterpret_cast<const double2 *>(base + (int64_t)(k + j) * a.e_stride));
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const double *cf = smc + (k + j) * 5;
      m0.x += cf[0] * v[j].x; m0.y += cf[0] * v[j].y;
      m1.x += cf[1] * v[j].x; m1.y += cf[1] * v[j].y;
      m2.x += cf[2] * v[j].x; m2.y += cf[2] * v[j].y;
      m3.x += cf[3] * v[j].x; m3.y += cf[3] * v[j].y;
      m4.x += cf[4] * v[j].x; m4.y += cf[4] * v[j].y;
    }
  }
  for (; k < nsys; ++k) {
    const double2 v = __ldcs(reinterpret_cast<const double2 *>(base + (int64_t)k * a.e_stride));
    const double *cf = smc + k * 5;
    m0.x += cf[0] * v.x; m0.y += cf[0] * v.y;
    m1.x += cf[1] * v.x; m1.y += cf[1] * v.y;
    m2.x += cf[2] * v.x; m2.y += cf[2] * v.y;
    m3.x += cf[3] * v.x; m3.y += cf[3] * v.y;
    m4.x += cf[4] * v.x; m4.y += cf[4] * v.y;
  }
  double *p = a.part + (size_t)c * 5 * a.e_stride + pos;
  *reinterpret_cast<double2 *>(p) = m0;
  *reinterpret_cast<double2 *>(p + a.e_stride) = m1;
  *reinterpret_cast<double2 *>(p + 2 * a.e_stride) = m2;
  *reinterpret_cast<double2 *>(p + 3 * a.e_stride) = m3;
  *reinterpret_cast<double2 *>(p + 4 * a.e_stride) = m4;
}

int nb_launch_moments_unstructured(nanobte_solver *h);

int nb_launch_moments(nanobte_solver *h) {
  if (h->brick) return 0;  // the partial moments came out of the sweep itself
  if (h->kind == 1) return nb_launch_moments_unstructured(h);
  MomentsArgs a;
  a.e = h->sw.e;
  a.mcoef = h->mcoef;
  a.part = h->part;
  a.e_stride = h->e_stride;
  int maxpos = 0, maxsys = 0;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) {
    a.cls_nsys[c] = h->cls_nsys[c];
    a.cls_row0[c] = h->cls_row0[c];
    a.cls_npos[c] = h->cls_npos[c];
    maxpos = max(maxpos, h->cls_npos[c]);
    maxsys = max(maxsys, h->cls_nsys[c]);
  }
  dim3 grid((maxpos + 511) / 512, h->n_cls);
  const size_t smem = (size_t)maxsys * 5 * sizeof(double);
  if (smem > 48 * 1024)
    NB_CUDA(h, cudaFuncSetAttribute(moments_structured_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  moments_structured_kernel<<<grid, 256, smem, h->stream>>>(a);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// =================================================================================================================
// (a6)/(a8) combine the class partials per cell (fixed class order), update T, track max |dT|, and refresh the
// sweep-order copies of theta.
// =================================================================================================================
struct UpdateArgs {
  int32_t n_act, n_cls, mode, dim;
  const double *part;
  int64_t e_stride;
  const int32_t *a2pos;  // [n_cls][n_act]
  double2 *tq[NB_MAX_CLASSES];
  double *theta, *theta_prev, *theta_SI, *theta_en, *q;
  const double *x;       // CG solution (mode 1)
  double beta, Csum;
  unsigned long long *maxdT;
  double *uns_theta;     // unstructured: nothing to permute (theta is read by cell id)
};

__global__ void __launch_bounds__(256) update_kernel(UpdateArgs u) {
  __shared__ double red[8];
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  double d = 0.0;
  if (a < u.n_act) {
    double th;
    if (u.mode == 0) {
      double m[5] = {0, 0, 0, 0, 0};
      for (int c = 0; c < u.n_cls; ++c) {
        const int64_t pos = u.a2pos[(size_t)c * u.n_act + a];
        const double *p = u.part + (size_t)c * 5 * u.e_stride + pos;
#pragma unroll
        for (int k = 0; k < 5; ++k) m[k] += p[(size_t)k * u.e_stride];
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
    for (int c = 0; c < u.n_cls; ++c) u.tq[c][u.a2pos[(size_t)c * u.n_act + a]].x = th;
  }
  d = warp_nanmax(d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = d;
  __syncthreads();
  if (threadIdx.x < 32) {
    d = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
    d = warp_nanmax(d);
    if (threadIdx.x == 0) atomicMax(u.maxdT, (unsigned long long)__double_as_longlong(d));
  }
}

int nb_launch_update_unstructured(nanobte_solver *h, int mode);

int nb_launch_update(nanobte_solver *h, int mode) {
  NB_CUDA(h, cudaMemsetAsync(h->d_maxdT, 0, sizeof(unsigned long long), h->stream));
  if (h->kind == 1) return nb_launch_update_unstructured(h, mode);
  if (h->brick) return nb_brick_update(h, mode);
  UpdateArgs u;
  u.n_act = h->n_act; u.n_cls = h->n_cls; u.mode = mode; u.dim = h->dim;
  u.part = h->part; u.e_stride = h->e_stride; u.a2pos = h->a2pos;
  for (int c = 0; c < NB_MAX_CLASSES; ++c) u.tq[c] = h->tq[c];
  u.theta = h->theta; u.theta_prev = h->theta_prev; u.theta_SI = h->theta_SI; u.theta_en = h->theta_en; u.q = h->q;
  u.x = h->cg_x; u.beta = h->beta; u.Csum = h->Csum; u.maxdT = h->d_maxdT; u.uns_theta = nullptr;
  update_kernel<<<(h->n_act + 255) / 256, 256, 0, h->stream>>>(u);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// ---- set_T: theta <- T - T_ref (cells -> active), refresh sweep-order copies --------------------------------------
__global__ void set_theta_kernel(int n_act, int n_cls, const int32_t *act2cell, const double *T, double T_ref,
                                 double *theta, const int32_t *a2pos, UpdateArgs u) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_act) return;
  const double th = T[act2cell[a]] - T_ref;
  theta[a] = th;
  for (int c = 0; c < n_cls; ++c) u.tq[c][a2pos[(size_t)c * n_act + a]].x = th;
}

int nb_launch_set_theta(nanobte_solver *h, const double *T_cells_dev) {
  if (h->brick) return nb_brick_set_theta(h, T_cells_dev);
  UpdateArgs u{};
  for (int c = 0; c < NB_MAX_CLASSES; ++c) u.tq[c] = h->tq[c];
  const int ncls = h->kind == 0 ? h->n_cls : 0;
  set_theta_kernel<<<(h->n_act + 255) / 256, 256, 0, h->stream>>>(h->n_act, ncls, h->act2cell, T_cells_dev, h->T_ref,
                                                                   h->theta, h->a2pos, u);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// ---- exports ---------------------------------------------------------------------------------------------------------
__global__ void scatter_cells_kernel(int n_cells, const int32_t *cell2act, const double *src, int src_stride,
                                     double *dst, int ncomp, double add) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cells) return;
  const int a = cell2act[c];
  for (int k = 0; k < ncomp; ++k) dst[(size_t)c * ncomp + k] = add + (a >= 0 ? src[(size_t)a * src_stride + k] : 0.0);
}

int nb_launch_scatter_cells(nanobte_solver *h, const double *src_act, double *dst_cells, int ncomp, double add) {
  const int stride = (src_act == h->q) ? 3 : 1;
  scatter_cells_kernel<<<(h->n_cells + 255) / 256, 256, 0, h->stream>>>(h->n_cells, h->cell2act, src_act, stride,
                                                                       dst_cells, ncomp, add);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

struct GetEArgs {
  int32_t n_cells, n_act, B, b0, nb, d0, nd, unstructured;
  const int32_t *cell2act, *a2pos, *dir_cls, *dir_row0;
  const double *e, *C;
  int64_t e_stride;
  double off_scale;  // T_ref / W, or 0 for the deviational export
  double *dst;
};

__global__ void get_e_kernel(GetEArgs g) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.n_cells) return;
  const int bi = blockIdx.y / g.nd, di = blockIdx.y % g.nd;
  const int b = g.b0 + bi, d = g.d0 + di;
  const int a = g.cell2act[c];
  double val = 0.0;
  if (a >= 0) {
    const int64_t pos = g.a2pos[(size_t)g.dir_cls[d] * g.n_act + a];
    val = g.unstructured ? g.e[((int64_t)d * g.e_stride + pos) * g.B + b] : g.e[((int64_t)g.dir_row0[d] + b) * g.e_stride + pos];
    val += g.C[b] * g.off_scale;
  }
  g.dst[((size_t)bi * g.nd + di) * g.n_cells + c] = val;
}

int nb_launch_get_e(nanobte_solver *h, int b0, int nb, int d0, int nd, double *dst_dev, int deviational) {
  if (nb == 0 || nd == 0) return 0;
  if (h->brick) return nb_brick_get_e(h, b0, nb, d0, nd, dst_dev, deviational);
  GetEArgs g;
  g.n_cells = h->n_cells; g.n_act = h->n_act; g.B = h->B; g.b0 = b0; g.nb = nb; g.d0 = d0; g.nd = nd;
  g.unstructured = h->kind;
  g.cell2act = h->cell2act; g.a2pos = h->a2pos; g.dir_cls = h->dir_cls; g.dir_row0 = h->bd.dir_row0; g.e = h->bd.e; g.C = h->bd.C;
  g.e_stride = h->e_stride; g.off_scale = deviational ? 0.0 : h->T_ref / h->W; g.dst = dst_dev;
  dim3 grid((h->n_cells + 255) / 256, nb * nd);
  get_e_kernel<<<grid, 256, 0, h->stream>>>(g);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// ---- boundary heat per tag (O8): one block per tag, fixed-order tree -----------------------------------------------------
__global__ void __launch_bounds__(256) tagheat_kernel(const int32_t *tagface_ptr, const int32_t *tagface, const double *faceflux,
                                                      const double *bf_area, int B, double *out) {
  __shared__ double red[256];
  const int t = blockIdx.x;
  double acc = 0.0;
  for (int k = tagface_ptr[t] + threadIdx.x; k < tagface_ptr[t + 1]; k += blockDim.x) {
    const int bf = tagface[k];
    double F = 0.0;
    for (int b = 0; b < B; ++b) F += faceflux[(size_t)bf * B + b];
    acc += bf_area[bf] * F;
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[t] = red[0];
}

int nb_launch_tagheat(nanobte_solver *h) {
  tagheat_kernel<<<h->n_tags, 256, 0, h->stream>>>(h->tagface_ptr, h->tagface, h->bd.faceflux, h->bd.bf_area, h->B, h->d_tagheat);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

// ---- band shards: the reflecting-face leak of R14c' summed over this solver's bands (nanobte_export_moments) -----------------------------
__global__ void leak_sum_kernel(int n_bf, int B, const double *faceflux, double *leak) {
  const int bf = blockIdx.x * blockDim.x + threadIdx.x;
  if (bf >= n_bf) return;
  double F = 0.0;
  for (int b = 0; b < B; ++b) F += faceflux[(size_t)bf * B + b];
  leak[bf] = F;
}

int nb_launch_leak_sum(nanobte_solver *h) {
  if (h->n_bf == 0) return 0;
  leak_sum_kernel<<<(h->n_bf + 255) / 256, 256, 0, h->stream>>>(h->n_bf, h->B, h->bd.faceflux, h->leak_sum);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}
