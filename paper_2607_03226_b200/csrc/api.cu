// api.cu -- the C-ABI entry points of libnanobte that do not depend on the mesh kind, plus the host-side
// validation and the upload of the tables both kinds share.  See include/nanobte.h for the contract.
#include <algorithm>
#include <numeric>
#include <cstdlib>

#include "brick.h"
#include "cg_mg.h"
#include "host_util.h"

int nb_fail(nanobte_solver *h, int code, const char *fmt, ...) {
  if (h) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    h->err = buf;
  }
  return code;
}

extern "C" const char *nanobte_strerror(int code) {
  switch (code) {
    case NANOBTE_OK: return "OK";
    case NANOBTE_NOT_CONVERGED: return "NOT_CONVERGED";
    case NANOBTE_E_INVALID: return "INVALID";
    case NANOBTE_E_ALLOC: return "ALLOC";
    case NANOBTE_E_CUDA: return "CUDA";
    case NANOBTE_E_ARCH: return "ARCH";
    case NANOBTE_E_UNTAGGED: return "UNTAGGED";
    case NANOBTE_E_SPECULAR: return "SPECULAR";
    case NANOBTE_E_CYCLE: return "CYCLE";
    case NANOBTE_E_QUADRATURE: return "QUADRATURE";
    case NANOBTE_E_SINGULAR: return "SINGULAR";
    case NANOBTE_E_NONFINITE: return "NONFINITE";
    case NANOBTE_E_UNSUPPORTED: return "UNSUPPORTED";
  }
  return "?";
}

extern "C" const char *nanobte_last_error(const nanobte_solver *h) { return h ? h->err.c_str() : "null handle"; }

int nb_check_device(nanobte_solver *h) {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n == 0)
    return nb_fail(h, NANOBTE_E_ARCH, "no CUDA device (%s); libnanobte has no CPU fallback",
                   e == cudaSuccess ? "count 0" : cudaGetErrorString(e));
  int dev = 0;
  cudaDeviceProp p;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&p, dev) != cudaSuccess)
    return nb_fail(h, NANOBTE_E_ARCH, "cannot query the CUDA device");
  if (p.major != 10) return nb_fail(h, NANOBTE_E_ARCH, "device is sm_%d%d; libnanobte is built for sm_100a only", p.major, p.minor);
  h->n_sm = p.multiProcessorCount;
  return 0;
}

// Host-side validation of the band table, the quadrature and the tag table, and the scalars derived from them:
//   W = sum_i w_i (Eq. 11), beta = sum_b C_b / tau_b (denominator of Eq. 5), sum_b C_b (R13),
//   source shares C_b / sum C (R5) and kappa_bulk (R14d).
// kappa_bulk is the kinetic conductivity with the isotropic part of the quadrature's second moment tensor
// M = sum_i w_i s_i s_i^T / W:  kappa = (trace of M over the mesh's own dimensions / dim) * sum_b C_b v_b^2 tau_b.
namespace {
struct AngularMoments {
  double zeroth = 0.0, first[3] = {0.0, 0.0, 0.0}, second_diag[3] = {0.0, 0.0, 0.0};
};
const char *check_bands(const nanobte_bands &t, int &bad) {
  for (bad = 0; bad < t.B; ++bad)
    if (!(t.C[bad] > 0.0 && t.v[bad] > 0.0 && t.tau[bad] > 0.0)) return "band %d: heat capacity, group velocity and relaxation time must all be positive";
  return nullptr;
}
}  // namespace

// Number of SMs of the current device if there is one (the plan built by workspace_bytes_* must match create's);
// leaves the default (148, B200) on a machine without a GPU, where only the host-side sizing runs.
void nb_query_sm_count(nanobte_solver *h) {
  int n = 0, dev = 0, sms = 0;
  if (cudaGetDeviceCount(&n) == cudaSuccess && n > 0 && cudaGetDevice(&dev) == cudaSuccess &&
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
    h->n_sm = sms;
  cudaGetLastError();
}

int nb_validate_common(nanobte_solver *h, int dim, const nanobte_bands *bands, const nanobte_quadrature *quad,
                       const nanobte_tag *tags, int n_tags, Common &c) {
  if (bands == nullptr || quad == nullptr) return nb_fail(h, NANOBTE_E_INVALID, "band table and quadrature are required");
  if (n_tags < 0 || (n_tags > 0 && tags == nullptr)) return nb_fail(h, NANOBTE_E_INVALID, "tag table missing");
  if (bands->B < 1 || bands->C == nullptr || bands->v == nullptr || bands->tau == nullptr)
    return nb_fail(h, NANOBTE_E_INVALID, "band table needs B >= 1 and the arrays C, v, tau");
  if (quad->D < 1 || quad->s == nullptr || quad->w == nullptr)
    return nb_fail(h, NANOBTE_E_INVALID, "quadrature needs D >= 1 and the arrays s, w");
  c.dim = dim;
  c.n_tags = n_tags;

  // tags first: cheapest, and independent of everything else
  c.tag_type.clear();
  c.tag_T.clear();
  for (int t = 0; t < n_tags; ++t) {
    const int ty = tags[t].type;
    if (ty != NANOBTE_THERMALIZING && ty != NANOBTE_DIFFUSE && ty != NANOBTE_SPECULAR && ty != NANOBTE_MIXED)
      return nb_fail(h, NANOBTE_E_INVALID, "tag %d has type %d; known types are 0..3", t, ty);
    c.tag_type.push_back(ty);
    c.tag_T.push_back(tags[t].T_wall);
  }

  // quadrature: unit vectors, positive weights, vanishing first moment (the T_ref part of q then drops out of Eq. 7)
  c.D = quad->D;
  c.s.assign(quad->s, quad->s + 3 * (size_t)c.D);
  c.w.assign(quad->w, quad->w + c.D);
  AngularMoments am;
  for (int i = 0; i < c.D; ++i) {
    const double wi = c.w[i], *si = &c.s[3 * (size_t)i];
    if (!(wi > 0.0)) return nb_fail(h, NANOBTE_E_QUADRATURE, "quadrature weight %d is %g; weights must be positive", i, wi);
    const double len2 = si[0] * si[0] + si[1] * si[1] + si[2] * si[2];
    if (std::fabs(std::sqrt(len2) - 1.0) > 1e-12) return nb_fail(h, NANOBTE_E_QUADRATURE, "direction %d has length %.15g, not 1", i, std::sqrt(len2));
    am.zeroth += wi;
    for (int a = 0; a < 3; ++a) {
      am.first[a] += wi * si[a];
      am.second_diag[a] += wi * si[a] * si[a];
    }
  }
  c.W = am.zeroth;
  for (int a = 0; a < dim; ++a)
    if (std::fabs(am.first[a]) > 1e-12 * c.W)
      return nb_fail(h, NANOBTE_E_QUADRATURE, "first angular moment does not vanish: sum_i w_i s_i[%d] = %g", a, am.first[a]);

  // bands
  c.B = bands->B;
  int bad = 0;
  if (const char *msg = check_bands(*bands, bad)) return nb_fail(h, NANOBTE_E_INVALID, msg, bad);
  c.C.assign(bands->C, bands->C + c.B);
  c.v.assign(bands->v, bands->v + c.B);
  c.tau.assign(bands->tau, bands->tau + c.B);
  c.Csum = std::accumulate(c.C.begin(), c.C.end(), 0.0);
  c.beta = 0.0;
  double cv2tau = 0.0;
  for (int b = 0; b < c.B; ++b) {
    c.beta += c.C[b] / c.tau[b];
    cv2tau += c.C[b] * c.v[b] * c.v[b] * c.tau[b];
  }
  c.share.resize(c.B);
  for (int b = 0; b < c.B; ++b) c.share[b] = bands->src_share != nullptr ? bands->src_share[b] : c.C[b] / c.Csum;
  double trace = 0.0;
  for (int a = 0; a < dim; ++a) trace += am.second_diag[a];
  c.kappa = cv2tau * trace / (dim * c.W);
  return 0;
}

int nb_find_mirror(const Common &c, int d, const double n[3]) {
  const double *s = &c.s[3 * d];
  const double sn = s[0] * n[0] + s[1] * n[1] + s[2] * n[2];
  const double r[3] = {s[0] - 2 * sn * n[0], s[1] - 2 * sn * n[1], s[2] - 2 * sn * n[2]};
  for (int j = 0; j < c.D; ++j) {
    const double d0 = c.s[3 * j] - r[0], d1 = c.s[3 * j + 1] - r[1], d2 = c.s[3 * j + 2] - r[2];
    if (d0 * d0 + d1 * d1 + d2 * d2 < 1e-18) return j;
  }
  return -1;
}

int nb_upload_generic(nanobte_solver *h, Arena &A, const Common &c, GenericTables &g) {
  const size_t na = g.act2cell.size(), nbf = g.bf_act.size();
  h->B = c.B; h->D = c.D; h->dim = c.dim; h->n_tags = c.n_tags;
  h->W = c.W; h->beta = c.beta; h->Csum = c.Csum; h->kappa = c.kappa;
  h->n_act = (int)na; h->n_bf = (int)nbf;
  h->h_C = c.C;
  BoundaryArgs &bd = h->bd;
  bd.n_bf = (int)nbf; bd.B = c.B; bd.D = c.D;
  bd.bf_act = A.put(g.bf_act);
  bd.bf_type = A.put(g.bf_type);
  bd.bf_p = A.put(g.bf_p);
  bd.bf_den = A.put(g.bf_den);
  bd.bf_area = A.put(g.bf_area);
  bd.bf_eps_w = A.put(g.bf_eps_w);
  bd.bf_sn = A.put(g.bf_sn);
  bd.bf_mirror = A.put(g.bf_mirror);
  bd.bf_inidx = A.put(g.bf_inidx);
  bd.bf_opos = A.put(g.bf_opos);
  bd.w = A.put(c.w);
  bd.C = A.put(c.C);
  bd.v = A.put(c.v);
  bd.dir_bin = A.put(g.dir_bin);
  bd.dir_nin = A.put(g.dir_nin);
  bd.dir_row0 = A.put(g.dir_row0);
  bd.bin = A.zeros<double>((size_t)g.bin_total);
  bd.G = A.zeros<double>(nbf * c.B);
  bd.faceflux = A.zeros<double>(nbf * c.B);
  h->n_inflow = 0;
  for (int d = 0; d < c.D; ++d) h->n_inflow += g.dir_nin[d];
  h->any_therm = false;
  for (size_t f = 0; f < nbf; ++f)
    if (g.bf_type[f] == NANOBTE_THERMALIZING) h->any_therm = true;
  h->mcoef = A.put(g.mcoef);
  h->act2cell = A.put(g.act2cell);
  h->cell2act = A.put(g.cell2act);
  h->vol = A.put(g.vol);
  h->Qdot = A.put(g.Qdot_act);
  h->theta = A.put(g.theta0);
  h->theta_prev = A.zeros<double>(na);
  h->theta_SI = A.zeros<double>(na);
  h->theta_en = A.zeros<double>(na);
  h->q = A.zeros<double>(na * 3);
  h->d_maxdT = A.zeros<unsigned long long>(4);
  // CG
  h->cg_nf = g.cg_nf;
  h->cg_nbr = A.put(g.cg_nbr);
  h->cg_coef = A.put(g.cg_coef);
  h->cg_diag = A.put(g.cg_diag);
  h->cellbf_ptr = A.put(g.cellbf_ptr);
  h->cellbf = A.put(g.cellbf);
  h->fourier_rhs = A.put(g.fourier_rhs);
  h->leak_sum = A.zeros<double>(nbf + 8);
  h->cg_x = A.zeros<double>(na);
  h->cg_r = A.zeros<double>(na);
  h->cg_p0 = A.zeros<double>(na);
  h->cg_p1 = A.zeros<double>(na);
  h->cg_rhs = A.zeros<double>(na);
  h->cg_scal = A.zeros<double>(16);
  h->cg_partial = A.zeros<double>(4 * 2048);
  // fused CG plan: the cells are renumbered so that every CTA owns a contiguous range that is also compact in space
  // (recursive coordinate bisection with prescribed part sizes: small halos); halo = neighbours owned by other CTAs
  {
    const int n = (int)na, nf = g.cg_nf;
    const int threads = 512;
    int nblk = std::max(1, std::min(h->n_sm, (n + 255) / 256));
    if (const char *env = std::getenv("NANOBTE_CG_NBLK"))  // test hook: fewer, larger chunks (more cells per thread) on small meshes
      nblk = std::max(1, std::min(nblk, std::atoi(env)));
    int chunk = (n + nblk - 1) / nblk;
    nblk = (n + chunk - 1) / chunk;
    const int cpt = chunk <= threads ? 1 : chunk <= 2 * threads ? 2 : chunk <= 4 * threads ? 4 : chunk <= 8 * threads ? 8 : 0;
    std::vector<int32_t> perm(n), inv(n);  // perm: CG index -> active index
    std::iota(perm.begin(), perm.end(), 0);
    if ((int)g.cg_xyz.size() == 3 * n && nblk > 1) {
      struct Job { int lo, hi, p0, p1; };
      std::vector<Job> stack{{0, n, 0, nblk}};
      while (!stack.empty()) {
        const Job J = stack.back();
        stack.pop_back();
        if (J.p1 - J.p0 <= 1) continue;
        double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
        for (int i = J.lo; i < J.hi; ++i)
          for (int k = 0; k < 3; ++k) {
            const double v = g.cg_xyz[3 * (size_t)perm[i] + k];
            mn[k] = std::min(mn[k], v);
            mx[k] = std::max(mx[k], v);
          }
        int ax = 0;
        for (int k = 1; k < 3; ++k) if (mx[k] - mn[k] > mx[ax] - mn[ax]) ax = k;
        const int pm = (J.p0 + J.p1) / 2;
        const int mid = std::min(J.hi, J.lo + (pm - J.p0) * chunk);  // parts p0..pm-1 are full chunks
        std::nth_element(perm.begin() + J.lo, perm.begin() + mid, perm.begin() + J.hi, [&](int32_t x, int32_t y) {
          const double vx = g.cg_xyz[3 * (size_t)x + ax], vy = g.cg_xyz[3 * (size_t)y + ax];
          return vx < vy || (vx == vy && x < y);
        });
        stack.push_back({J.lo, mid, J.p0, pm});
        stack.push_back({mid, J.hi, pm, J.p1});
      }
      for (int k = 0; k < nblk; ++k)  // deterministic, memory-friendly order inside a chunk
        std::sort(perm.begin() + k * chunk, perm.begin() + std::min(n, (k + 1) * chunk));
    }
    for (int i = 0; i < n; ++i) inv[perm[i]] = i;
    std::vector<double> coef_p((size_t)nf * n), diag_p(n);
    std::vector<int32_t> nbr_p((size_t)nf * n);
    for (int i = 0; i < n; ++i) {
      diag_p[i] = g.cg_diag[perm[i]];
      for (int f = 0; f < nf; ++f) {
        coef_p[(size_t)f * n + i] = g.cg_coef[(size_t)f * n + perm[i]];
        nbr_p[(size_t)f * n + i] = inv[g.cg_nbr[(size_t)f * n + perm[i]]];
      }
    }
    // face-uniform stencil (uniform structured grids): every face slot has one coefficient value, or none
    bool uni = nf <= 6;
    double cfu[6] = {0, 0, 0, 0, 0, 0};
    for (int f = 0; f < nf && uni; ++f)
      for (int i = 0; i < n && uni; ++i) {
        const double c = coef_p[(size_t)f * n + i];
        if (c == 0.0) continue;
        if (cfu[f] == 0.0) cfu[f] = c;
        uni = cfu[f] == c;
      }
    if (std::getenv("NANOBTE_CG_NO_UNI")) uni = false;  // test hook: the general stencil path
    std::vector<int32_t> nloc((size_t)nf * n), hptr(nblk + 1, 0), hidx;
    int nh_cap = 0;
    for (int k = 0; k < nblk; ++k) {
      const int a0 = k * chunk, a1 = std::min(n, a0 + chunk);
      std::vector<int32_t> halo;
      for (int i = a0; i < a1; ++i)
        for (int f = 0; f < nf; ++f) {
          const int j = nbr_p[(size_t)f * n + i];
          if (coef_p[(size_t)f * n + i] != 0.0 && (j < a0 || j >= a1)) halo.push_back(j);
        }
      std::sort(halo.begin(), halo.end());
      halo.erase(std::unique(halo.begin(), halo.end()), halo.end());
      for (int i = a0; i < a1; ++i)
        for (int f = 0; f < nf; ++f) {
          const int j = nbr_p[(size_t)f * n + i];
          int32_t loc = i - a0;  // faces without a neighbour carry coefficient 0 and point at the cell itself
          if (coef_p[(size_t)f * n + i] != 0.0)
            loc = (j >= a0 && j < a1) ? j - a0 : chunk + (int32_t)(std::lower_bound(halo.begin(), halo.end(), j) - halo.begin());
          nloc[(size_t)f * n + i] = loc;
        }
      hidx.insert(hidx.end(), halo.begin(), halo.end());
      hptr[k + 1] = (int32_t)hidx.size();
      nh_cap = std::max(nh_cap, (int)halo.size());
    }
    h->cgf_perm = A.put(perm);
    h->cgf_coef = A.put(coef_p);
    h->cgf_diag = A.put(diag_p);
    nh_cap += 1;  // one more slot that is in nobody's halo: stays zero
    if (uni)      // a missing neighbour reads the zero slot (its coefficient is the face's, not 0)
      for (int i = 0; i < n; ++i)
        for (int f = 0; f < nf; ++f)
          if (coef_p[(size_t)f * n + i] == 0.0) nloc[(size_t)f * n + i] = chunk + nh_cap - 1;
    h->cgf_uni = uni;
    for (int f = 0; f < 6; ++f) h->cgf_cfu[f] = cfu[f];
    h->cgf_nblk = nblk; h->cgf_chunk = chunk; h->cgf_cpt = cpt; h->cgf_nh_cap = nh_cap;
    h->cgf_smem = (3 * (size_t)chunk + 2 * (size_t)nh_cap) * sizeof(double) + (size_t)nh_cap * sizeof(int32_t) + 1024;
    h->cgf_ok = cpt > 0 && chunk + nh_cap < 65536 && (nf == 3 || nf == 4 || nf == 6) && h->cgf_smem <= 200 * 1024;
    h->cg_force_generic = std::getenv("NANOBTE_CG_GENERIC") != nullptr;  // test hook: the multi-pass fallback kernel
    h->cgf_nloc = A.put(nloc);
    h->cgf_hptr = A.put(hptr);
    h->cgf_hidx = A.put(hidx);
    h->cgf_w = A.zeros<double>(2 * na);
    h->cgf_part = A.zeros<double>((size_t)4 * nblk + 8);
    h->cgf_bar = A.zeros<unsigned int>(4);
    h->cgf_xprev = A.zeros<double>(2 * na);
    h->cgf_gpart = A.zeros<double>((size_t)8 * nblk + 8);
    h->cgf_recycle = std::getenv("NANOBTE_CG_NO_RECYCLE") == nullptr;
    // uniform 3-D structured grids: multigrid-preconditioned CG (cg_mg.cu) unless a test hook asks for a plain-CG kernel
    if (uni && nf == 6 && c.dim == 3 && g.cg_grid[0] > 0 && !h->cg_force_generic && std::getenv("NANOBTE_CG_NO_MG") == nullptr &&
        std::getenv("NANOBTE_CG_NO_UNI") == nullptr && std::getenv("NANOBTE_CG_NO_RECYCLE") == nullptr) {
      // the coefficients in the order of the faces, before the CG renumbering
      double cfu0[6] = {0, 0, 0, 0, 0, 0};
      for (int f = 0; f < 6; ++f) cfu0[f] = cfu[f];
      const int rc_mg = nb_mg_build(h, A, g, cfu0, g.cg_grid);
      if (rc_mg < 0) return rc_mg;
    }
  }
  h->tagface_ptr = A.put(g.tagface_ptr);
  h->tagface = A.put(g.tagface);
  h->d_tagheat = A.zeros<double>((size_t)std::max(1, c.n_tags));
  return A.rc;
}

// ---------------------------------------------------------------------------------------------------------------
extern "C" void nanobte_destroy(nanobte_solver *h) {
  if (!h) return;
  if (h->stream || h->arena) cudaStreamSynchronize(h->stream);
  nb_free_unstructured(h);
  nb_free_brick(h);
  nb_free_mg(h);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->aux_stream) cudaStreamDestroy(h->aux_stream);
  if (h->arena && h->arena_owned) cudaFree(h->arena);
  if (h->h_pinned) cudaFreeHost(h->h_pinned);
  delete h;
}

// One transport sweep.  keep_e = 0 lets the tile-dataflow sweep leave the distribution on chip (moments and wall values
// are all the iteration needs); the other sweeps always store it.
static int sweep_internal(nanobte_solver *h, int keep_e) {
  h->swept_since_closure = true;
  h->therm_stale = true;
  if (h->brick) return nb_launch_sweep_brick(h, keep_e);
  return h->kind == 0 ? nb_launch_sweep_structured(h) : nb_launch_sweep_unstructured(h);
}

extern "C" int nanobte_sweep(nanobte_solver *h) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  return sweep_internal(h, h->keep_e ? 1 : 0);
}

extern "C" int nanobte_set_keep_e(nanobte_solver *h, int32_t keep) {
  if (!h) return NANOBTE_E_INVALID;
  h->keep_e = keep != 0;
  return 0;
}

static int read_maxdT(nanobte_solver *h, double *out) {
  // d_maxdT[0] = bit pattern of max|dT| (non-negative double), d_maxdT[1] = CG iteration count of the last solve
  NB_CUDA(h, cudaMemcpyAsync(h->h_pinned, h->d_maxdT, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  NB_CUDA(h, cudaStreamSynchronize(h->stream));
  *out = h->h_pinned[0];
  return std::isfinite(*out) ? 0 : nb_fail(h, NANOBTE_E_NONFINITE, "max|dT| is not finite");
}

extern "C" int nanobte_update_temperature(nanobte_solver *h, double *max_dT) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  int rc;
  const bool fork = h->brick && h->swept_since_closure && h->aux_stream;
  if (fork) {  // O4 + O5 beside the closures (disjoint data: partial moments / theta here, wall rows / G / inflow rows there)
    NB_CUDA(h, cudaEventRecord(h->ev_fork, h->stream));
    NB_CUDA(h, cudaStreamWaitEvent(h->aux_stream, h->ev_fork, 0));
    cudaStream_t main = h->stream;
    h->stream = h->aux_stream;
    rc = nb_launch_moments(h);
    if (rc >= 0) rc = nb_launch_update(h, 0);
    h->stream = main;
    if (rc < 0) return rc;
    NB_CUDA(h, cudaEventRecord(h->ev_join, h->aux_stream));
  }
  if (h->swept_since_closure) {  // G, face fluxes, inflow cache for the next sweep (O3); once per sweep
    if ((rc = nb_launch_boundary(h)) < 0) return rc;
    h->swept_since_closure = false;
  }
  if (fork) {
    NB_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_join, 0));
  } else {
    if ((rc = nb_launch_moments(h)) < 0) return rc;   // O4
    if ((rc = nb_launch_update(h, 0)) < 0) return rc; // O5
  }
  h->leak_imported = false;  // a correction after this update sums its own bands' face fluxes unless moments are imported
  if (max_dT) return read_maxdT(h, max_dT);
  return 0;
}

extern "C" int nanobte_diffusion_correct(nanobte_solver *h, int32_t *cg_iters, double *max_dT) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  if (!h->any_therm) return nb_fail(h, NANOBTE_E_SINGULAR, "synthetic mode needs at least one thermalizing face");
  int rc;
  if ((rc = nb_cg_solve(h, nullptr)) < 0) return rc;
  if ((rc = nb_launch_update(h, 1)) < 0) return rc;
  double d = 0;
  if ((rc = read_maxdT(h, &d)) < 0) return rc;
  unsigned long long it;
  memcpy(&it, h->h_pinned + 1, sizeof(it));
  const bool cg_failed = (it >> 40) & 1ull;  // the CG kernels flag "stopped on cg_max_iter above the tolerance"
  if (cg_iters) *cg_iters = (int32_t)(it & 0xffffffffull);
  if (max_dT) *max_dT = d;
  if (cg_failed) {
    h->cgf_nprev = 0;  // do not recycle a solution that is not one
    nb_fail(h, NANOBTE_NOT_CONVERGED, "CG stopped at cg_max_iter = %d above rtol = %g", h->cg_max_iter, h->cg_rtol);
    return NANOBTE_NOT_CONVERGED;
  }
  return 0;
}

// ---- band shards (Eq. 14): this shard's terms of the update out, the sums over all shards in ---------------------------
// The sums a shard needs about the WHOLE band table: out[0] = beta, out[1] = sum C, out[2] = kappa (same code as create).
extern "C" int nanobte_band_totals(const nanobte_bands *bands, const nanobte_quadrature *quad, int32_t dim, double *out) {
  if (!out || (dim != 2 && dim != 3)) return NANOBTE_E_INVALID;
  nanobte_solver tmp;
  Common c;
  const int rc = nb_validate_common(&tmp, dim, bands, quad, nullptr, 0, c);
  if (rc < 0) return rc;
  out[0] = c.beta; out[1] = c.Csum; out[2] = c.kappa;
  return 0;
}

extern "C" int64_t nanobte_moments_len(const nanobte_solver *h) { return h ? (int64_t)5 * h->n_act + h->n_bf : 0; }

extern "C" int nanobte_export_moments(nanobte_solver *h, double *dst, int32_t dst_is_device) {
  if (!h || !h->arena || !dst) return NANOBTE_E_INVALID;
  const size_t na = (size_t)h->n_act;
  const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  int rc = nb_launch_leak_sum(h);  // leak_sum[bf] = sum over this shard's bands of the face flux (R14c')
  if (rc < 0) return rc;
  NB_CUDA(h, cudaMemcpyAsync(dst, h->theta_SI, na * sizeof(double), kind, h->stream));
  NB_CUDA(h, cudaMemcpyAsync(dst + na, h->theta_en, na * sizeof(double), kind, h->stream));
  NB_CUDA(h, cudaMemcpyAsync(dst + 2 * na, h->q, 3 * na * sizeof(double), kind, h->stream));
  if (h->n_bf) NB_CUDA(h, cudaMemcpyAsync(dst + 5 * na, h->leak_sum, (size_t)h->n_bf * sizeof(double), kind, h->stream));
  if (!dst_is_device) NB_CUDA(h, cudaStreamSynchronize(h->stream));
  return 0;
}

extern "C" int nanobte_import_moments(nanobte_solver *h, const double *src, int32_t src_is_device, double *max_dT) {
  if (!h || !h->arena || !src) return NANOBTE_E_INVALID;
  const size_t na = (size_t)h->n_act;
  const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  NB_CUDA(h, cudaMemcpyAsync(h->theta_SI, src, na * sizeof(double), kind, h->stream));
  NB_CUDA(h, cudaMemcpyAsync(h->theta_en, src + na, na * sizeof(double), kind, h->stream));
  NB_CUDA(h, cudaMemcpyAsync(h->q, src + 2 * na, 3 * na * sizeof(double), kind, h->stream));
  if (h->n_bf) NB_CUDA(h, cudaMemcpyAsync(h->leak_sum, src + 5 * na, (size_t)h->n_bf * sizeof(double), kind, h->stream));
  h->leak_imported = true;
  // T <- T_SI (Eq. 6) and max|T_new - T_old| through the update kernel's "T_SI + delta" form with delta = 0
  NB_CUDA(h, cudaMemsetAsync(h->cg_x, 0, na * sizeof(double), h->stream));
  int rc = nb_launch_update(h, 1);
  if (rc < 0) return rc;
  if (max_dT) return read_maxdT(h, max_dT);
  return 0;
}

extern "C" int nanobte_init_fourier(nanobte_solver *h, int32_t *cg_iters) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  if (!h->any_therm) return nb_fail(h, NANOBTE_E_SINGULAR, "the Fourier guess needs at least one thermalizing face");
  // R21: A theta = V Qdot + sum_thermalizing kappa A_f (T_w - T_ref) / d_cf with the operator of the synthetic
  // correction; the right-hand side is a table built at create, the solver is the CG of nanobte_diffusion_correct
  h->cgf_nprev = 0;
  h->cg_rhs_direct = h->fourier_rhs;
  int rc = nb_cg_solve(h, nullptr);
  h->cg_rhs_direct = nullptr;
  h->cgf_nprev = 0;  // this solution says nothing about the corrections to come
  if (rc < 0) return rc;
  if ((rc = nb_launch_scatter_cells(h, h->cg_x, h->part, 1, h->T_ref)) < 0) return rc;
  if ((rc = nb_launch_set_theta(h, h->part)) < 0) return rc;
  NB_CUDA(h, cudaMemcpyAsync(h->h_pinned, h->d_maxdT, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  NB_CUDA(h, cudaStreamSynchronize(h->stream));
  unsigned long long it;
  memcpy(&it, h->h_pinned + 1, sizeof(it));
  if (cg_iters) *cg_iters = (int32_t)(it & 0xffffffffull);
  if ((it >> 40) & 1ull) {
    nb_fail(h, NANOBTE_NOT_CONVERGED, "CG stopped at cg_max_iter = %d above rtol = %g", h->cg_max_iter, h->cg_rtol);
    return NANOBTE_NOT_CONVERGED;
  }
  return 0;
}

extern "C" int nanobte_solve(nanobte_solver *h, double tol, int32_t max_iter, int32_t mode, int32_t *iters_out,
                             double *last_dT_out) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  if (mode != 0 && mode != 1) return nb_fail(h, NANOBTE_E_INVALID, "mode must be 0 (plain) or 1 (synthetic)");
  if (mode == 1 && !h->any_therm) return nb_fail(h, NANOBTE_E_SINGULAR, "synthetic mode needs at least one thermalizing face");
  h->hist_dT.clear();
  h->hist_cg.clear();
  h->cgf_nprev = 0;  // a solve never depends on what the handle did before (recycled CG guesses start afresh)
  double dT = INFINITY;
  int n = 0, rc = NANOBTE_NOT_CONVERGED, r;
  bool cg_failed = false;
  while (n < max_iter) {
    int cg = 0;
    if ((r = sweep_internal(h, 0)) < 0) return r;
    if (mode == 0) {
      if ((r = nanobte_update_temperature(h, &dT)) < 0) return r;
    } else {
      if ((r = nanobte_update_temperature(h, nullptr)) < 0) return r;
      if ((r = nanobte_diffusion_correct(h, &cg, &dT)) < 0) return r;
      cg_failed = r == NANOBTE_NOT_CONVERGED;
    }
    ++n;
    h->hist_dT.push_back(dT);
    h->hist_cg.push_back(cg);
    if (dT < tol) {
      rc = cg_failed ? NANOBTE_NOT_CONVERGED : NANOBTE_OK;  // an outer iterate built on an unconverged CG is not a converged state
      break;
    }
  }
  if (iters_out) *iters_out = n;
  if (last_dT_out) *last_dT_out = dT;
  return rc;
}

extern "C" int nanobte_step(nanobte_solver *h, int32_t mode, double *max_dT, int32_t *cg_iters) {
  if (!h || !h->arena) return NANOBTE_E_INVALID;
  if (mode != 0 && mode != 1) return nb_fail(h, NANOBTE_E_INVALID, "mode must be 0 (plain) or 1 (synthetic)");
  if (mode == 1 && !h->any_therm) return nb_fail(h, NANOBTE_E_SINGULAR, "synthetic mode needs at least one thermalizing face");
  int r;
  double dT = 0.0;
  if ((r = sweep_internal(h, 0)) < 0) return r;
  if (cg_iters) *cg_iters = 0;
  if (mode == 0) {
    r = nanobte_update_temperature(h, &dT);
  } else {
    if ((r = nanobte_update_temperature(h, nullptr)) < 0) return r;
    r = nanobte_diffusion_correct(h, cg_iters, &dT);
  }
  if (max_dT) *max_dT = dT;
  return r;
}

// ---- getters / setters ---------------------------------------------------------------------------------------
// Device scratch for getters that need a host round trip: the part[] buffer (>= 5 * e_stride doubles) is free
// between update_temperature calls; it always holds at least 3 * n_cells doubles (checked at create).
static int copy_out(nanobte_solver *h, const double *dev_src, double *dst, size_t n, int dst_is_device) {
  if (dst_is_device) {
    NB_CUDA(h, cudaMemcpyAsync(dst, dev_src, n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  } else {
    NB_CUDA(h, cudaMemcpyAsync(dst, dev_src, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    NB_CUDA(h, cudaStreamSynchronize(h->stream));
  }
  return 0;
}

extern "C" int nanobte_set_T(nanobte_solver *h, const double *T, int32_t src_is_device) {
  if (!h || !h->arena || !T) return NANOBTE_E_INVALID;
  const double *src = T;
  if (!src_is_device) {
    NB_CUDA(h, cudaMemcpyAsync(h->part, T, (size_t)h->n_cells * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    src = h->part;
  }
  int rc = nb_launch_set_theta(h, src);
  if (rc < 0) return rc;
  if (!src_is_device) NB_CUDA(h, cudaStreamSynchronize(h->stream));
  return 0;
}

extern "C" int nanobte_get_T(nanobte_solver *h, int32_t which, double *dst, int32_t dst_is_device) {
  if (!h || !h->arena || !dst) return NANOBTE_E_INVALID;
  const double *src = which == 0 ? h->theta : which == 1 ? h->theta_en : which == 2 ? h->theta_SI : nullptr;
  if (!src) return nb_fail(h, NANOBTE_E_INVALID, "which must be 0, 1 or 2");
  double *stage = dst_is_device ? dst : h->part;
  int rc = nb_launch_scatter_cells(h, src, stage, 1, h->T_ref);
  if (rc < 0) return rc;
  if (!dst_is_device) return copy_out(h, stage, dst, (size_t)h->n_cells, 0);
  return 0;
}

extern "C" int nanobte_get_q(nanobte_solver *h, double *dst, int32_t dst_is_device) {
  if (!h || !h->arena || !dst) return NANOBTE_E_INVALID;
  double *stage = dst_is_device ? dst : h->part;
  int rc = nb_launch_scatter_cells(h, h->q, stage, h->dim, 0.0);
  if (rc < 0) return rc;
  if (!dst_is_device) return copy_out(h, stage, dst, (size_t)h->n_cells * h->dim, 0);
  return 0;
}

extern "C" int nanobte_get_e(nanobte_solver *h, int32_t b0, int32_t nb, int32_t d0, int32_t nd, double *dst,
                             int32_t deviational, int32_t dst_is_device) {
  if (!h || !h->arena || !dst) return NANOBTE_E_INVALID;
  if (b0 < 0 || nb < 0 || b0 + nb > h->B || d0 < 0 || nd < 0 || d0 + nd > h->D)
    return nb_fail(h, NANOBTE_E_INVALID, "band/direction range");
  if (h->brick && !h->brick->e_valid) {  // the last sweep kept the distribution on chip: sweep once more, storing it
    int rc = sweep_internal(h, 1);
    if (rc < 0) return rc;
  }
  if (dst_is_device) return nb_launch_get_e(h, b0, nb, d0, nd, dst, deviational);
  // host destination: one (band, direction) row at a time through the part[] scratch
  for (int b = 0; b < nb; ++b)
    for (int d = 0; d < nd; ++d) {
      int rc = nb_launch_get_e(h, b0 + b, 1, d0 + d, 1, h->part, deviational);
      if (rc < 0) return rc;
      rc = copy_out(h, h->part, dst + ((size_t)b * nd + d) * h->n_cells, (size_t)h->n_cells, 0);
      if (rc < 0) return rc;
    }
  return 0;
}

extern "C" int nanobte_get_G(nanobte_solver *h, double *dst, int32_t dst_is_device) {
  if (!h || !h->arena || !dst) return NANOBTE_E_INVALID;
  int rc = nb_refresh_thermalizing(h);
  if (rc < 0) return rc;
  return copy_out(h, h->bd.G, dst, (size_t)h->n_bf * h->B, dst_is_device);
}

extern "C" int nanobte_get_boundary_heat(nanobte_solver *h, double *per_tag) {
  if (!h || !h->arena || !per_tag) return NANOBTE_E_INVALID;
  if (h->n_tags == 0) return 0;
  int rc = nb_refresh_thermalizing(h);
  if (rc < 0) return rc;
  rc = nb_launch_tagheat(h);
  if (rc < 0) return rc;
  return copy_out(h, h->d_tagheat, per_tag, (size_t)h->n_tags, 0);
}

extern "C" int nanobte_get_history(nanobte_solver *h, double *dT, int32_t *cg_iters, int32_t cap) {
  if (!h) return NANOBTE_E_INVALID;
  const int n = std::min<int>((int)h->hist_dT.size(), cap);
  for (int k = 0; k < n; ++k) {
    if (dT) dT[k] = h->hist_dT[k];
    if (cg_iters) cg_iters[k] = h->hist_cg[k];
  }
  return (int)h->hist_dT.size();
}

extern "C" int nanobte_get_info(const nanobte_solver *h, nanobte_info *o) {
  if (!h || !o) return NANOBTE_E_INVALID;
  o->dim = h->dim; o->n_cells = h->n_cells; o->n_active = h->n_act; o->B = h->B; o->D = h->D; o->n_bfaces = h->n_bf;
  o->n_octants = h->n_cls; o->n_planes = h->n_planes; o->n_tasks = h->n_tasks; o->sweep_G = h->sweep_G;
  o->sweep_threads = h->sweep_threads; o->sweep_rmax = h->sweep_rmax; o->pencil_axis = h->pencil_axis; o->n_pos = h->n_pos;
  o->n_inflow = h->n_inflow; o->device_bytes = h->arena_bytes; o->sweep_smem_bytes = h->sweep_smem;
  const bool fused = h->cgf_ok && !h->cg_force_generic;
  o->cg_fused = fused; o->cg_cells_per_thread = fused ? h->cgf_cpt : 0; o->cg_ctas = fused ? h->cgf_nblk : h->cg_blocks;
  o->cg_face_uniform = fused && h->cgf_uni; o->cg_recycle = fused && h->cgf_recycle;
  o->cg_multigrid = h->mg && !h->cg_force_generic ? 1 : 0;
  o->cg_mg_levels = o->cg_multigrid ? h->mg->levels : 0;
  o->sweep_variant = h->kind == 1 ? 1 : h->sweep_variant;
  return 0;
}

extern "C" int64_t nanobte_launch_count(const nanobte_solver *h) { return h ? h->launches : 0; }
extern "C" double nanobte_kappa(const nanobte_solver *h) { return h ? h->kappa : 0.0; }
