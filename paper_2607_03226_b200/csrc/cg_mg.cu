// cg_mg.cu -- (a7) synthetic correction on uniform 3-D structured grids: conjugate gradient preconditioned by one
// aggregation-multigrid V-cycle, the whole solve in ONE cooperative launch (one CTA per SM).
//
//   A delta = rhs,  stop at ||r|| <= rtol ||rhs||      (Eq. 8-12; readings R14a-e as in cg.cu)
//
// The paper solves this system with a cached sparse LU; the oracle with an unpreconditioned CG from
// zero (R14e).  Here the system and the stopping rule are the oracle's, the iterates are not (reading R14e'): on config 4
// the plain CG needs ~570 iterations of one grid barrier each, this one 11-16 iterations of ~41 us without any.
//
// Hierarchy (built at create, nb_mg_build): level l+1 = 2 x 2 x 2 aggregates of the level-l lattice, piecewise-constant
// prolongation P, Galerkin operators P^T A P.  On a uniform grid every fine face of direction f has the coefficient
// cfu[f], so a coarse face is a COUNT of fine faces and the coarse diagonal is the counts plus the summed Dirichlet terms:
// the coarse operators are exact and cost two bytes per face.
//   levels 0..2  distributed: a CTA owns whole level-3 aggregates (8^3 cells) and the octree below them, so restriction and
//                prolongation never leave the CTA; iterates cross CTA borders through global memory, tagged (mg_tag below).
//   levels 3..   a few hundred unknowns: every CTA holds them in shared memory and repeats the same arithmetic
//                (bitwise identical, no communication); the coarsest level (<= 32 unknowns) is a dense inverse.
// Smoother: x <- x + B (g - A x) with B = two damped-Jacobi steps on the CTA's own diagonal block (no communication),
//   B = (w1 + w2) D^-1 - w1 w2 D^-1 A_own D^-1,  w1 = 1.45, w2 = 0.65:
// symmetric whatever the weights, and positive definite because the eigenvalues of D^-1 A_own lie in (0, 2) and
// 1/w1 + 1/w2 = 2.23 > 2.  Two different weights put the roots of the error polynomial (1 - w1 z)(1 - w2 z) at both ends of
// the rough part of the spectrum (a Chebyshev smoother of degree two) instead of twice in its middle: 20 % fewer CG
// iterations than w1 = w2 = 0.9 at the same cost.  Once before and once after the coarse correction, which is scaled by
// tau = 1.9 (over-correction for the piecewise-constant prolongation).  The V-cycle is a fixed symmetric positive definite
// operator, as CG requires.
// CG in the Chronopoulos-Gear form (one reduction per iteration): u = M^-1 r, w = A u, gamma = (r,u), delta = (w,u).
// All reductions are fixed trees over per-CTA partials: bitwise reproducible, identical scalars in every CTA.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "cg_mg.h"

namespace {

constexpr unsigned long long kCgNotConverged = 1ull << 40;  // as in cg.cu

__device__ __forceinline__ void grid_barrier(unsigned int *bar, unsigned int target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned int v;
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
    } while (v < target);
  }
  __syncthreads();
}

// Values that cross CTA borders carry a sequence bit in their last mantissa bit (a relative perturbation of at most
// 2.2e-16, deterministic): the value is its own ready flag.  Buffers are double-buffered by iteration parity and zeroed
// before the launch; iteration `it` writes buffer it & 1 with bit ((it >> 1) & 1) ^ 1, so what is left in that buffer from
// iteration it - 2 (or the zeros of the launch) has the other bit.  A CTA cannot be two iterations ahead of a CTA it
// exchanges with (every iteration ends in an all-to-all of the dot products), which is what makes two buffers enough.
__device__ __forceinline__ double mg_tag(double x, unsigned bit) {
  return __hiloint2double(__double2hiint(x), (int)(((unsigned)__double2loint(x) & ~1u) | bit));
}
__device__ __forceinline__ double mg_load(const double *p, unsigned bit) {
  double v;
  for (;;) {
    asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    if ((((unsigned)__double2loint(v)) & 1u) == bit) return v;
    __nanosleep(20);
  }
}

#ifdef MG_PROF
__device__ unsigned long long g_mg_prof[16];
#define MGP(k) do { if (tid == 0 && blockIdx.x == 0) { const long long t_ = clock64(); g_mg_prof[k] += (unsigned long long)(t_ - tprof); tprof = t_; } } while (0)
#else
#define MGP(k)
#endif

// A level held in shared memory (levels 1.. ; level 0 keeps its stencil in registers).
struct Lv {
  int n;                 // own unknowns
  double *x;             // [n + halo (+1)] iterate
  double *g, *res, *tmp; // [n]
  const uint16_t *nbr, *cnt;  // [6][stride]
  const double *dinv, *diag;  // [n]
  int stride;
};

__device__ __forceinline__ double apply_full(const Lv &L, const double *v, int i, const double *cfu) {
  double acc = L.diag[i] * v[i];
#pragma unroll
  for (int f = 0; f < 6; ++f) acc -= (double)L.cnt[f * L.stride + i] * cfu[f] * v[L.nbr[f * L.stride + i]];
  return acc;
}
// own diagonal block only: neighbours outside the CTA's own range do not exist
__device__ __forceinline__ double apply_own(const Lv &L, const double *v, int i, const double *cfu) {
  double acc = L.diag[i] * v[i];
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    const int j = L.nbr[f * L.stride + i];
    if (j < L.n) acc -= (double)L.cnt[f * L.stride + i] * cfu[f] * v[j];
  }
  return acc;
}

// x = B g with x = 0 before (two Jacobi steps on the own block); leaves x[0..n).  Two block-synchronised phases.
__device__ __forceinline__ void presmooth(const Lv &L, const double *cfu, const double rho) {
  const int tid = threadIdx.x;
  for (int i = tid; i < L.n; i += kMgThreads) L.tmp[i] = L.dinv[i] * L.g[i];
  __syncthreads();
  for (int i = tid; i < L.n; i += kMgThreads) L.x[i] = L.tmp[i] + rho * L.dinv[i] * (L.g[i] - apply_own(L, L.tmp, i, cfu));
  __syncthreads();
}
// res = g - A x (halo of x valid)
__device__ __forceinline__ void residual(const Lv &L, const double *cfu) {
  for (int i = threadIdx.x; i < L.n; i += kMgThreads) L.res[i] = L.g[i] - apply_full(L, L.x, i, cfu);
  __syncthreads();
}
// x += B (g - A x)   (halo of x valid; the halo is not updated).  Two block-synchronised phases.
__device__ __forceinline__ void postsmooth(const Lv &L, const double *cfu, const double rho) {
  const int tid = threadIdx.x;
  for (int i = tid; i < L.n; i += kMgThreads) {
    const double r = L.g[i] - apply_full(L, L.x, i, cfu);
    L.res[i] = r;
    L.tmp[i] = L.dinv[i] * r;
  }
  __syncthreads();
  for (int i = tid; i < L.n; i += kMgThreads)
    L.x[i] += L.tmp[i] + rho * L.dinv[i] * (L.res[i] - apply_own(L, L.tmp, i, cfu));
  __syncthreads();
}

template <int CPT>
__global__ void __launch_bounds__(kMgThreads, 1) cg_mg_kernel(const MgArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, k = blockIdx.x;
  const int a3lo = a.a3ptr[k], na3 = a.a3ptr[k + 1] - a3lo;
  const int n0 = na3 * 512, n1 = na3 * 64, n2 = na3 * 8;
  const int64_t base0 = (int64_t)a3lo * 512, base1 = (int64_t)a3lo * 64, base2 = (int64_t)a3lo * 8;
  const int h0lo = a.hptr[0][k], nh0 = a.hptr[0][k + 1] - h0lo;
  const int h1lo = a.hptr[1][k], nh1 = a.hptr[1][k + 1] - h1lo;
  const int h2lo = a.hptr[2][k], nh2 = a.hptr[2][k + 1] - h2lo;
  double cfu[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) cfu[f] = a.cfu[f];

  // ---- shared memory ----------------------------------------------------------------------------------------------------------------
  unsigned char *sp = smem_raw;
  auto take_d = [&](int n) { double *p = reinterpret_cast<double *>(sp); sp += (size_t)((n + 1) & ~1) * 8; return p; };
  auto take_h = [&](int n) { uint16_t *p = reinterpret_cast<uint16_t *>(sp); sp += (size_t)((n + 7) & ~7) * 2; return p; };
  auto take_i = [&](int n) { int32_t *p = reinterpret_cast<int32_t *>(sp); sp += (size_t)((n + 3) & ~3) * 4; return p; };
  double *xs = take_d(a.cap0);                    // CG solution
  double *ps = take_d(a.cap0);                    // CG search direction
  double *x0 = take_d(a.cap0 + a.caph0 + 2);      // level-0 iterate of the V-cycle / u, with halo and the zero slot
  double *y0 = take_d(a.cap0);                    // level-0 scratch (residual for the restriction, Jacobi exchange)
  Lv L1, L2;
  L1.n = n1; L1.stride = a.cap1;
  L1.x = take_d(a.cap1 + a.caph1 + 2); L1.g = take_d(a.cap1); L1.res = take_d(a.cap1); L1.tmp = take_d(a.cap1);
  double *dinv1 = take_d(a.cap1), *diag1 = take_d(a.cap1);
  L2.n = n2; L2.stride = a.cap2;
  L2.x = take_d(a.cap2 + a.caph2 + 2); L2.g = take_d(a.cap2); L2.res = take_d(a.cap2); L2.tmp = take_d(a.cap2);
  double *dinv2 = take_d(a.cap2), *diag2 = take_d(a.cap2);
  double *gx = take_d(a.ntot), *gg = take_d(a.ntot), *gres = take_d(a.ntot), *gtmp = take_d(a.ntot);
  double *gdinv = take_d(a.ntot), *gdiag = take_d(a.ntot);
  const int nc = a.n_l[a.nlev - 1];
  double *ginv = take_d(nc * nc);
  double *red = take_d(64);
  int32_t *hidx0 = take_i(a.caph0), *hidx1 = take_i(a.caph1), *hidx2 = take_i(a.caph2);
  int32_t *hpar0 = take_i(a.caph0), *hpar1 = take_i(a.caph1), *hpar2 = take_i(a.caph2);
  uint16_t *nbr1 = take_h(6 * a.cap1), *cnt1 = take_h(6 * a.cap1), *nbr2 = take_h(6 * a.cap2), *cnt2 = take_h(6 * a.cap2);
  uint16_t *gnbr = take_h(6 * a.ntot), *gcnt = take_h(6 * a.ntot), *gchild = take_h(8 * a.ntot), *gpar = take_h(a.ntot);
  L1.nbr = nbr1; L1.cnt = cnt1; L1.dinv = dinv1; L1.diag = diag1;
  L2.nbr = nbr2; L2.cnt = cnt2; L2.dinv = dinv2; L2.diag = diag2;

#ifdef MG_PROF
  long long tprof = clock64();
  const long long tprof0 = tprof;
#endif
  // ---- load the CTA's tables ------------------------------------------------------------------------------------------------------------
  for (int i = tid; i < n1; i += kMgThreads) {
    dinv1[i] = a.dinv[1][base1 + i]; diag1[i] = a.diag[1][base1 + i];
    for (int f = 0; f < 6; ++f) {
      nbr1[f * a.cap1 + i] = a.nbr[1][(int64_t)f * a.a3ptr[a.nblk] * 64 + base1 + i];
      cnt1[f * a.cap1 + i] = a.cnt[1][(int64_t)f * a.a3ptr[a.nblk] * 64 + base1 + i];
    }
  }
  for (int i = tid; i < n2; i += kMgThreads) {
    dinv2[i] = a.dinv[2][base2 + i]; diag2[i] = a.diag[2][base2 + i];
    for (int f = 0; f < 6; ++f) {
      nbr2[f * a.cap2 + i] = a.nbr[2][(int64_t)f * a.a3ptr[a.nblk] * 8 + base2 + i];
      cnt2[f * a.cap2 + i] = a.cnt[2][(int64_t)f * a.a3ptr[a.nblk] * 8 + base2 + i];
    }
  }
  for (int i = tid; i < a.ntot; i += kMgThreads) {
    gdinv[i] = a.gdinv[i]; gdiag[i] = a.gdiag[i]; gpar[i] = a.gpar[i];
    for (int f = 0; f < 6; ++f) { gnbr[f * a.ntot + i] = a.gnbr[f * a.ntot + i]; gcnt[f * a.ntot + i] = a.gcnt[f * a.ntot + i]; }
    for (int c = 0; c < 8; ++c) gchild[c * a.ntot + i] = a.gchild[c * a.ntot + i];
  }
  for (int i = tid; i < nc * nc; i += kMgThreads) ginv[i] = a.ginv[i];
  for (int j = tid; j < nh0; j += kMgThreads) { hidx0[j] = a.hidx[0][h0lo + j]; hpar0[j] = a.hpar[0][h0lo + j]; }
  for (int j = tid; j < nh1; j += kMgThreads) { hidx1[j] = a.hidx[1][h1lo + j]; hpar1[j] = a.hpar[1][h1lo + j]; }
  for (int j = tid; j < nh2; j += kMgThreads) { hidx2[j] = a.hidx[2][h2lo + j]; hpar2[j] = a.hpar[2][h2lo + j]; }
  if (tid == 0) { x0[n0 + nh0] = 0.0; L1.x[n1 + nh1] = 0.0; L2.x[n2 + nh2] = 0.0; }

  MGP(11);
  // ---- level 0: stencil, right-hand side (R14c, R14c'), CG vectors ------------------------------------------------------------------------
  const int64_t nslot0 = (int64_t)a.a3ptr[a.nblk] * 512;
  uint16_t nl[CPT][6];
  double dv[CPT], dg[CPT], r[CPT], s[CPT], w[CPT];
  int cell[CPT];
#pragma unroll
  for (int c = 0; c < CPT; ++c) {
    const int li = tid + c * kMgThreads;
    dv[c] = 0.0; dg[c] = 1.0; r[c] = s[c] = w[c] = 0.0; cell[c] = -1;
#pragma unroll
    for (int f = 0; f < 6; ++f) nl[c][f] = (uint16_t)(n0 + nh0);
    if (li < n0) {
      xs[li] = ps[li] = 0.0;
      dv[c] = a.dinv0[base0 + li]; dg[c] = a.diag0[base0 + li]; cell[c] = a.cell0[base0 + li];
#pragma unroll
      for (int f = 0; f < 6; ++f) nl[c][f] = a.nbr0[(int64_t)f * nslot0 + base0 + li];
      const int io = cell[c];
      if (io >= 0) {
        double rhs;
        if (a.rhs_direct) {
          rhs = a.rhs_direct[io];
        } else {
          rhs = a.vol[io] * a.beta * (a.theta_SI[io] - a.theta_prev[io]);  // R14c
          for (int q = a.cellbf_ptr[io]; q < a.cellbf_ptr[io + 1]; ++q) {  // R14c'
            const int bf = a.cellbf[q];
            double F = 0.0;
            if (a.leak_sum) F = a.leak_sum[bf];
            else for (int b = 0; b < a.B; ++b) F += a.faceflux[(size_t)bf * a.B + b];
            rhs += a.bf_area[bf] * F;
          }
        }
        r[c] = rhs;
      }
    }
  }
  __syncthreads();
  MGP(12);

  auto A0 = [&](int c, const double *v, double vc) {  // full operator, row of slot c of this thread
    double acc = dg[c] * vc;
#pragma unroll
    for (int f = 0; f < 6; ++f) acc -= cfu[f] * v[nl[c][f]];
    return acc;
  };
  auto A0own = [&](int c, const double *v, double vc) {  // own diagonal block
    double acc = dg[c] * vc;
#pragma unroll
    for (int f = 0; f < 6; ++f) {
      const int j = nl[c][f];
      if (j < n0) acc -= cfu[f] * v[j];
    }
    return acc;
  };
  int it = 0;
  // publish the own part of an iterate, then read the halo: no barrier (see mg_tag)
  auto exchange = [&](double *xg2, int64_t nslot, int64_t base, const double *xv, int n, double *halo, const int32_t *hidx, int nh) {
    double *buf = xg2 + (size_t)(it & 1) * nslot;
    const unsigned bit = ((unsigned)(it >> 1) & 1u) ^ 1u;
    for (int i = tid; i < n; i += kMgThreads) __stcg(buf + base + i, mg_tag(xv[i], bit));
    for (int j = tid; j < nh; j += kMgThreads) halo[j] = mg_load(buf + hidx[j], bit);
    __syncthreads();
  };

  unsigned int epoch = 1;
  // ---- recycled initial guess: x_0 = Galerkin projection of the right-hand side on the span of the last two solutions (the operator
  // never changes and successive corrections become collinear; cg.cu has the same step).  Their halo values were written by
  // earlier launches and are simply read; one reduction of six scalars.  The stopping rule keeps ||rhs||.
  double bb_total = -1.0;
  if (a.nprev > 0) {
    double X[2][CPT], AX[2][CPT];
#pragma unroll
    for (int v = 0; v < 2; ++v) {
      const double *xp = a.xprev + (size_t)v * nslot0;
      const bool have = v < a.nprev;
      __syncthreads();
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const int li = tid + c * kMgThreads;
        X[v][c] = (have && li < n0) ? xp[base0 + li] : 0.0;
        if (li < n0) x0[li] = X[v][c];
      }
      for (int j = tid; j < nh0; j += kMgThreads) x0[n0 + j] = have ? xp[hidx0[j]] : 0.0;
      __syncthreads();
#pragma unroll
      for (int c = 0; c < CPT; ++c) AX[v][c] = A0(c, x0, X[v][c]);
    }
    double sums[6] = {0, 0, 0, 0, 0, 0};  // X1.b, X2.b, X1.AX1, X1.AX2, X2.AX2, b.b
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      sums[0] += X[0][c] * r[c];
      sums[1] += X[1][c] * r[c];
      sums[2] += X[0][c] * AX[0][c];
      sums[3] += X[0][c] * AX[1][c];
      sums[4] += X[1][c] * AX[1][c];
      sums[5] += r[c] * r[c];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 6; ++q) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sums[q] += __shfl_xor_sync(0xffffffffu, sums[q], o);
      if (lane == 0) y0[q * (kMgThreads / 32) + wid] = sums[q];
    }
    __syncthreads();
    if (tid < 6) {
      double t = 0.0;
      for (int w2 = 0; w2 < kMgThreads / 32; ++w2) t += y0[tid * (kMgThreads / 32) + w2];
      a.gpart[(size_t)k * 8 + tid] = t;
    }
    grid_barrier(a.bar, epoch++ * a.nblk);
    double tot[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      double t = 0.0;
      for (int c2 = lane; c2 < a.nblk; c2 += 32) t += __ldcg(a.gpart + (size_t)c2 * 8 + q);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      tot[q] = t;
    }
    bb_total = tot[5];
    double c1 = 0.0, c2 = 0.0;
    const double det = tot[2] * tot[4] - tot[3] * tot[3];
    if (a.nprev > 1 && det > 1e-8 * tot[2] * tot[4]) {  // two independent directions
      c1 = (tot[0] * tot[4] - tot[1] * tot[3]) / det;
      c2 = (tot[1] * tot[2] - tot[0] * tot[3]) / det;
    } else if (tot[2] > 0.0) {
      c1 = tot[0] / tot[2];
    }
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      if (li < n0) {
        xs[li] = c1 * X[0][c] + c2 * X[1][c];
        r[c] -= c1 * AX[0][c] + c2 * AX[1][c];
      }
    }
    __syncthreads();
  }
  double g_prev = 1.0, alpha_prev = 1.0, stop2 = 0.0;
  bool not_converged = false;
  const int64_t nslot1 = (int64_t)a.a3ptr[a.nblk] * 64, nslot2 = (int64_t)a.a3ptr[a.nblk] * 8;
  MGP(13);
  for (;; ++it) {
    const unsigned bit = ((unsigned)(it >> 1) & 1u) ^ 1u;
    MGP(9);
    // =================================== u = M^-1 r : one V-cycle ===================================================================
    // ---- level 0 down: x = B r, exchange, residual, restriction
    double xv[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      xv[c] = dv[c] * r[c];
      if (li < n0) y0[li] = xv[c];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      xv[c] += a.rho * dv[c] * (r[c] - A0own(c, y0, xv[c]));
      if (li < n0) x0[li] = xv[c];
    }
    __syncthreads();
    exchange(a.xg[0], nslot0, base0, x0, n0, x0 + n0, hidx0, nh0);
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      if (li < n0) y0[li] = r[c] - A0(c, x0, xv[c]);
    }
    __syncthreads();
    for (int i = tid; i < n1; i += kMgThreads) {
      const double *q = y0 + 8 * i;
      L1.g[i] = ((q[0] + q[1]) + (q[2] + q[3])) + ((q[4] + q[5]) + (q[6] + q[7]));
    }
    __syncthreads();
    MGP(0);
    // ---- level 1 down
    presmooth(L1, cfu, a.rho);
    exchange(a.xg[1], nslot1, base1, L1.x, n1, L1.x + n1, hidx1, nh1);
    residual(L1, cfu);
    for (int i = tid; i < n2; i += kMgThreads) {
      const double *q = L1.res + 8 * i;
      L2.g[i] = ((q[0] + q[1]) + (q[2] + q[3])) + ((q[4] + q[5]) + (q[6] + q[7]));
    }
    __syncthreads();
    MGP(1);
    // ---- level 2 down; the level-3 right-hand side is published
    presmooth(L2, cfu, a.rho);
    exchange(a.xg[2], nslot2, base2, L2.x, n2, L2.x + n2, hidx2, nh2);
    residual(L2, cfu);
    {
      double *g3b = a.g3 + (size_t)(it & 1) * a.n_l[3];
      for (int i = tid; i < na3; i += kMgThreads) {
        const double *q = L2.res + 8 * i;
        __stcg(g3b + a3lo + i, mg_tag(((q[0] + q[1]) + (q[2] + q[3])) + ((q[4] + q[5]) + (q[6] + q[7])), bit));
      }
      for (int i = tid; i < a.n_l[3]; i += kMgThreads) gg[i] = mg_load(g3b + i, bit);
      __syncthreads();
    }
    MGP(2);
    // ---- levels 3.. : the same arithmetic in every CTA
    for (int l = 3; l < a.nlev; ++l) {
      const int o = a.off_l[l], n = a.n_l[l];
      Lv G;
      G.n = n; G.x = gx + o; G.g = gg + o; G.res = gres + o; G.tmp = gtmp + o; G.nbr = gnbr + o; G.cnt = gcnt + o;
      G.dinv = gdinv + o; G.diag = gdiag + o; G.stride = a.ntot;
      if (l == a.nlev - 1) {  // dense inverse
        for (int i = tid; i < n; i += kMgThreads) {
          double acc = 0.0;
          for (int j = 0; j < n; ++j) acc += ginv[i * n + j] * G.g[j];
          G.x[i] = acc;
        }
        __syncthreads();
        break;
      }
      presmooth(G, cfu, a.rho);
      residual(G, cfu);
      const int o2 = a.off_l[l + 1], n2c = a.n_l[l + 1];
      for (int i = tid; i < n2c; i += kMgThreads) {
        double acc = 0.0;
        for (int c = 0; c < 8; ++c) {
          const uint16_t ch = gchild[c * a.ntot + o2 + i];
          if (ch != 0xffffu) acc += G.res[ch];
        }
        gg[o2 + i] = acc;
      }
      __syncthreads();
    }
    for (int l = a.nlev - 2; l >= 3; --l) {
      const int o = a.off_l[l], n = a.n_l[l], o2 = a.off_l[l + 1];
      Lv G;
      G.n = n; G.x = gx + o; G.g = gg + o; G.res = gres + o; G.tmp = gtmp + o; G.nbr = gnbr + o; G.cnt = gcnt + o;
      G.dinv = gdinv + o; G.diag = gdiag + o; G.stride = a.ntot;
      for (int i = tid; i < n; i += kMgThreads) G.x[i] += a.tau * gx[o2 + gpar[o + i]];
      __syncthreads();
      postsmooth(G, cfu, a.rho);
    }
    MGP(3);
    // ---- level 2 up: correction of own and halo entries from level 3 (every CTA has all of it), post-smoothing, publish
    for (int i = tid; i < n2; i += kMgThreads)
      if (dinv2[i] != 0.0) L2.x[i] += a.tau * gx[a3lo + (i >> 3)];  // empty slots stay zero
    for (int j = tid; j < nh2; j += kMgThreads) L2.x[n2 + j] += a.tau * gx[hpar2[j]];
    __syncthreads();
    postsmooth(L2, cfu, a.rho);
    exchange(a.xu[2], nslot2, base2, L2.x, n2, L2.x + n2, hidx2, nh2);
    MGP(4);
    // ---- level 1 up
    for (int i = tid; i < n1; i += kMgThreads)
      if (dinv1[i] != 0.0) L1.x[i] += a.tau * L2.x[i >> 3];
    for (int j = tid; j < nh1; j += kMgThreads) L1.x[n1 + j] += a.tau * L2.x[hpar1[j]];
    __syncthreads();
    postsmooth(L1, cfu, a.rho);
    exchange(a.xu[1], nslot1, base1, L1.x, n1, L1.x + n1, hidx1, nh1);
    MGP(5);
    // ---- level 0 up: correction, x += B (r - A x); the result is u
    for (int j = tid; j < nh0; j += kMgThreads) x0[n0 + j] += a.tau * L1.x[hpar0[j]];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      if (li < n0) {
        if (dv[c] != 0.0) xv[c] += a.tau * L1.x[li >> 3];  // empty slots stay zero
        x0[li] = xv[c];
      }
    }
    __syncthreads();
    double rs[CPT], y1[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      rs[c] = r[c] - A0(c, x0, xv[c]);
      y1[c] = dv[c] * rs[c];
      if (li < n0) y0[li] = y1[c];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      xv[c] += y1[c] + a.rho * dv[c] * (rs[c] - A0own(c, y0, y1[c]));  // u
      if (li < n0) x0[li] = xv[c];
    }
    __syncthreads();
    MGP(6);
    // =================================== w = A u, the three dot products =============================================================
    exchange(a.xu[0], nslot0, base0, x0, n0, x0 + n0, hidx0, nh0);
    double gam = 0.0, del = 0.0, rho = 0.0;
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      w[c] = A0(c, x0, xv[c]);
      gam += r[c] * xv[c];
      del += w[c] * xv[c];
      rho += r[c] * r[c];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      gam += __shfl_xor_sync(0xffffffffu, gam, o);
      del += __shfl_xor_sync(0xffffffffu, del, o);
      rho += __shfl_xor_sync(0xffffffffu, rho, o);
    }
    if (lane == 0) { red[3 * wid] = gam; red[3 * wid + 1] = del; red[3 * wid + 2] = rho; }
    __syncthreads();
    double *pp = a.part + (size_t)(it & 1) * a.nblk * 4;
    if (wid == 0) {
      double G = lane < kMgThreads / 32 ? red[3 * lane] : 0.0, D = lane < kMgThreads / 32 ? red[3 * lane + 1] : 0.0,
             R = lane < kMgThreads / 32 ? red[3 * lane + 2] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        G += __shfl_xor_sync(0xffffffffu, G, o);
        D += __shfl_xor_sync(0xffffffffu, D, o);
        R += __shfl_xor_sync(0xffffffffu, R, o);
      }
      if (lane == 0) { __stcg(pp + 4 * k, mg_tag(G, bit)); __stcg(pp + 4 * k + 1, mg_tag(D, bit)); __stcg(pp + 4 * k + 2, mg_tag(R, bit)); }
      // every CTA reads the tagged partials of every CTA (the same values, bit for bit) and sums them in a fixed order
      G = 0.0; D = 0.0; R = 0.0;
      for (int q = lane; q < a.nblk; q += 32) {
        G += mg_load(pp + 4 * q, bit);
        D += mg_load(pp + 4 * q + 1, bit);
        R += mg_load(pp + 4 * q + 2, bit);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        G += __shfl_xor_sync(0xffffffffu, G, o);
        D += __shfl_xor_sync(0xffffffffu, D, o);
        R += __shfl_xor_sync(0xffffffffu, R, o);
      }
      if (lane == 0) { red[60] = G; red[61] = D; red[62] = R; }
    }
    __syncthreads();
    gam = red[60]; del = red[61]; rho = red[62];
    __syncthreads();
    MGP(7);
#ifdef MG_PROF
    if (tid == 0 && blockIdx.x == 0) g_mg_prof[10] += 1;
#endif
    if (it == 0) stop2 = a.rtol * a.rtol * (bb_total >= 0.0 ? bb_total : rho);  // without a guess x_0 = 0: r_0 = rhs
    if (!(rho > stop2)) break;
    if (it >= a.max_iter) { not_converged = true; break; }
    const double bet = it ? gam / g_prev : 0.0;
    const double alpha = it ? gam / (del - bet * gam / alpha_prev) : gam / del;
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kMgThreads;
      if (li < n0) {
        const double pc = fma(bet, ps[li], xv[c]);
        ps[li] = pc;
        s[c] = fma(bet, s[c], w[c]);
        xs[li] = fma(alpha, pc, xs[li]);
        r[c] = fma(-alpha, s[c], r[c]);
      }
    }
    g_prev = gam;
    alpha_prev = alpha;
  }
#pragma unroll
  for (int c = 0; c < CPT; ++c) {
    const int li = tid + c * kMgThreads;
    if (li < n0) {
      if (cell[c] >= 0) a.x[cell[c]] = xs[li];
      a.xprev[nslot0 + base0 + li] = a.xprev[base0 + li];  // history of the recycled initial guess
      a.xprev[base0 + li] = xs[li];
    }
  }
  if (k == 0 && tid == 0) *a.iters_out = (unsigned long long)it | (not_converged ? kCgNotConverged : 0ull);
#ifdef MG_PROF
  if (tid == 0 && blockIdx.x == 0) { g_mg_prof[14] += (unsigned long long)(clock64() - tprof0); g_mg_prof[15] += 1; }
#endif
}

typedef void (*mg_fn)(MgArgs);
mg_fn mg_pick(int cpt) {
  switch (cpt) {
    case 1: return cg_mg_kernel<1>;
    case 2: return cg_mg_kernel<2>;
    case 3: return cg_mg_kernel<3>;
    case 4: return cg_mg_kernel<4>;
    case 5: return cg_mg_kernel<5>;
    case 6: return cg_mg_kernel<6>;
    case 7: return cg_mg_kernel<7>;
    case 8: return cg_mg_kernel<8>;
  }
  return nullptr;
}

// ---- host: the lattice of one level ---------------------------------------------------------------------------------------------------------
struct Lat {
  int d[3] = {0, 0, 0};
  std::vector<uint8_t> act;
  std::vector<int32_t> cnt[6];
  std::vector<double> dir;     // summed Dirichlet (thermalizing-face) terms
  std::vector<int32_t> id;     // unknown / slot number, -1 = none
  size_t size() const { return (size_t)d[0] * d[1] * d[2]; }
  size_t at(int i, int j, int k) const { return (size_t)i + (size_t)d[0] * ((size_t)j + (size_t)d[1] * k); }
};

// inverse of a small symmetric positive definite matrix (Gauss-Jordan with partial pivoting); false if singular
bool dense_inverse(std::vector<double> &M, int n) {
  std::vector<double> I((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) I[(size_t)i * n + i] = 1.0;
  for (int c = 0; c < n; ++c) {
    int p = c;
    for (int r2 = c + 1; r2 < n; ++r2)
      if (std::fabs(M[(size_t)r2 * n + c]) > std::fabs(M[(size_t)p * n + c])) p = r2;
    if (!(std::fabs(M[(size_t)p * n + c]) > 0.0)) return false;
    if (p != c)
      for (int j = 0; j < n; ++j) { std::swap(M[(size_t)p * n + j], M[(size_t)c * n + j]); std::swap(I[(size_t)p * n + j], I[(size_t)c * n + j]); }
    const double inv = 1.0 / M[(size_t)c * n + c];
    for (int j = 0; j < n; ++j) { M[(size_t)c * n + j] *= inv; I[(size_t)c * n + j] *= inv; }
    for (int r2 = 0; r2 < n; ++r2) {
      if (r2 == c) continue;
      const double f = M[(size_t)r2 * n + c];
      if (f == 0.0) continue;
      for (int j = 0; j < n; ++j) { M[(size_t)r2 * n + j] -= f * M[(size_t)c * n + j]; I[(size_t)r2 * n + j] -= f * I[(size_t)c * n + j]; }
    }
  }
  M.swap(I);
  return true;
}

}  // namespace

// Builds the hierarchy and the per-CTA tables.  Returns 0 and leaves h->mg == nullptr when the plan does not fit (the caller
// keeps the plain fused CG); < 0 only on an allocation error.
int nb_mg_build(nanobte_solver *h, Arena &A, const GenericTables &g, const double *cfu, const int grid[3]) {
  const int na = (int)g.act2cell.size();
  if (g.cg_nf != 6 || na < 64) return 0;
  // Jacobi weights and over-correction, scanned on configs 3 and 4, on cuts and on grids with 4:2:1 spacings (CG iterations per
  // solve on config 4 after the first few source iterations: 17.8 at 0.9 / 0.9 / 2.0, 14.2 at 1.45 / 0.65 / 1.9; the count
  // rises steeply once 1/w1 + 1/w2 comes within 0.1 of 2, e.g. 23 at 1.4 / 0.75)
  double omega = 1.45, omega2 = 0.65, tau = 1.9;
  if (const char *env = std::getenv("NANOBTE_MG_OMEGA")) { omega = std::atof(env); omega2 = omega; }  // tuning hooks
  if (const char *env = std::getenv("NANOBTE_MG_OMEGA2")) omega2 = std::atof(env);
  if (const char *env = std::getenv("NANOBTE_MG_TAU")) tau = std::atof(env);
  // ---- lattices -------------------------------------------------------------------------------------------------------------------------------
  std::vector<Lat> lat(1);
  {
    Lat &L = lat[0];
    for (int k = 0; k < 3; ++k) L.d[k] = grid[k];
    L.act.assign(L.size(), 0); L.dir.assign(L.size(), 0.0); L.id.assign(L.size(), -1);
    for (int f = 0; f < 6; ++f) L.cnt[f].assign(L.size(), 0);
    for (int a = 0; a < na; ++a) {
      const int i = (int)g.cg_xyz[3 * (size_t)a], j = (int)g.cg_xyz[3 * (size_t)a + 1], k = (int)g.cg_xyz[3 * (size_t)a + 2];
      const size_t p = L.at(i, j, k);
      L.act[p] = 1; L.id[p] = a;
      double off = 0.0;
      for (int f = 0; f < 6; ++f) {
        const double c = g.cg_coef[(size_t)f * na + a];
        if (c != 0.0) {
          if (c != cfu[f]) return 0;  // not face-uniform after all
          L.cnt[f][p] = 1;
          off += c;
        }
      }
      const double dir = g.cg_diag[a] - off;
      L.dir[p] = dir > 1e-13 * g.cg_diag[a] ? dir : 0.0;
    }
  }
  int nlev = 1;
  for (;;) {
    const Lat &F = lat.back();
    int nact = 0;
    for (uint8_t v : F.act) nact += v;
    if (nlev >= 4 && (nact <= kMgCoarsest || (F.d[0] == 1 && F.d[1] == 1 && F.d[2] == 1))) break;
    if (nlev >= kMgMaxLevels) return 0;
    Lat C;
    for (int k = 0; k < 3; ++k) C.d[k] = (F.d[k] + 1) / 2;
    C.act.assign(C.size(), 0); C.dir.assign(C.size(), 0.0); C.id.assign(C.size(), -1);
    for (int f = 0; f < 6; ++f) C.cnt[f].assign(C.size(), 0);
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          if (!F.act[p]) continue;
          const size_t q = C.at(i >> 1, j >> 1, k >> 1);
          C.act[q] = 1;
          C.dir[q] += F.dir[p];
          const int co[3] = {i, j, k};
          for (int f = 0; f < 6; ++f)
            if ((co[f >> 1] & 1) == (f & 1)) C.cnt[f][q] += F.cnt[f][p];  // the child sits on that side of its aggregate
        }
    lat.push_back(std::move(C));
    ++nlev;
  }
  if (nlev < 4) return 0;
  const int nc = [&] { int n = 0; for (uint8_t v : lat[nlev - 1].act) n += v; return n; }();
  if (nc > kMgCoarsest || nc < 1) return 0;
  for (int l = 1; l < nlev; ++l)
    for (int f = 0; f < 6; ++f)
      for (int32_t v : lat[l].cnt[f]) if (v > 65535) return 0;

  // ---- level-3 aggregates -> CTAs (recursive coordinate bisection with prescribed part sizes) ----------------------------------------------
  Lat &L3 = lat[3];
  std::vector<int32_t> agg;  // lattice positions of the active level-3 cells
  for (size_t p = 0; p < L3.size(); ++p) if (L3.act[p]) agg.push_back((int32_t)p);
  const int n3 = (int)agg.size();
  int nblk = std::max(1, std::min(h->n_sm, n3));
  if (const char *env = std::getenv("NANOBTE_CG_NBLK")) nblk = std::max(1, std::min(nblk, std::atoi(env)));
  std::vector<int32_t> a3ptr(nblk + 1, 0);
  for (int k = 0; k < nblk; ++k) a3ptr[k + 1] = a3ptr[k] + n3 / nblk + (k < n3 % nblk ? 1 : 0);
  {
    auto coord = [&](int32_t p, int ax) { return ax == 0 ? p % L3.d[0] : ax == 1 ? (p / L3.d[0]) % L3.d[1] : p / (L3.d[0] * L3.d[1]); };
    struct Job { int lo, hi, p0, p1; };
    std::vector<Job> stack{{0, n3, 0, nblk}};
    while (!stack.empty()) {
      const Job J = stack.back();
      stack.pop_back();
      if (J.p1 - J.p0 <= 1) continue;
      int mn[3] = {1 << 30, 1 << 30, 1 << 30}, mx[3] = {-1, -1, -1};
      for (int i = J.lo; i < J.hi; ++i)
        for (int ax = 0; ax < 3; ++ax) { mn[ax] = std::min(mn[ax], coord(agg[i], ax)); mx[ax] = std::max(mx[ax], coord(agg[i], ax)); }
      int ax = 0;
      for (int q = 1; q < 3; ++q) if (mx[q] - mn[q] > mx[ax] - mn[ax]) ax = q;
      const int pm = (J.p0 + J.p1) / 2, mid = J.lo + (a3ptr[pm] - a3ptr[J.p0]);
      std::nth_element(agg.begin() + J.lo, agg.begin() + mid, agg.begin() + J.hi, [&](int32_t x, int32_t y) {
        const int cx = coord(x, ax), cy = coord(y, ax);
        return cx < cy || (cx == cy && x < y);
      });
      stack.push_back({J.lo, mid, J.p0, pm});
      stack.push_back({mid, J.hi, pm, J.p1});
    }
    for (int k = 0; k < nblk; ++k) std::sort(agg.begin() + a3ptr[k], agg.begin() + a3ptr[k + 1]);
  }
  std::vector<int32_t> owner3(n3);
  for (int k = 0; k < nblk; ++k)
    for (int a = a3ptr[k]; a < a3ptr[k + 1]; ++a) { L3.id[agg[a]] = a; owner3[a] = k; }
  int amax = 0;
  for (int k = 0; k < nblk; ++k) amax = std::max(amax, a3ptr[k + 1] - a3ptr[k]);
  const int cpt = (amax * 512 + kMgThreads - 1) / kMgThreads;
  if (cpt > 8) return 0;
  // slots of levels 2, 1: id = parent's id * 8 + child code
  for (int l = 2; l >= 1; --l) {
    Lat &F = lat[l];
    const Lat &P = lat[l + 1];
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          F.id[p] = F.act[p] ? P.id[P.at(i >> 1, j >> 1, k >> 1)] * 8 + (((k & 1) << 2) | ((j & 1) << 1) | (i & 1)) : -1;
        }
  }
  // level-0 slots need both numbers: slot0[lattice] and the active index (lat[0].id)
  std::vector<int32_t> slot0(lat[0].size(), -1);
  {
    const Lat &F = lat[0], &P = lat[1];
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          if (!F.act[p]) continue;
          slot0[p] = P.id[P.at(i >> 1, j >> 1, k >> 1)] * 8 + (((k & 1) << 2) | ((j & 1) << 1) | (i & 1));
        }
  }
  // levels >= 4: compressed lattice order
  std::vector<int32_t> n_l(nlev, 0);
  n_l[3] = n3;
  for (int l = 4; l < nlev; ++l) {
    int n = 0;
    for (size_t p = 0; p < lat[l].size(); ++p) if (lat[l].act[p]) lat[l].id[p] = n++;
    n_l[l] = n;
  }
  for (int l = 3; l < nlev; ++l) if (n_l[l] > 65534) return 0;

  // ---- distributed levels: stencils in local indices, halo lists -----------------------------------------------------------------------------
  const int64_t nslot[3] = {(int64_t)n3 * 512, (int64_t)n3 * 64, (int64_t)n3 * 8};
  const int shift[3] = {9, 6, 3};  // slot >> shift = level-3 aggregate
  auto slot_of = [&](int l, size_t p) -> int32_t { return l == 0 ? slot0[p] : lat[l].id[p]; };
  std::vector<std::vector<int32_t>> halo[3];   // per level, per CTA: sorted global slots
  for (int l = 0; l < 3; ++l) halo[l].assign(nblk, {});
  const int dx[6] = {-1, 1, 0, 0, 0, 0}, dy[6] = {0, 0, -1, 1, 0, 0}, dz[6] = {0, 0, 0, 0, -1, 1};
  for (int l = 0; l < 3; ++l) {
    const Lat &F = lat[l];
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          if (!F.act[p]) continue;
          const int me = owner3[slot_of(l, p) >> shift[l]];
          for (int f = 0; f < 6; ++f) {
            if (F.cnt[f][p] == 0) continue;
            const size_t q = F.at(i + dx[f], j + dy[f], k + dz[f]);
            const int32_t sq = slot_of(l, q);
            if (owner3[sq >> shift[l]] != me) halo[l][me].push_back(sq);
          }
        }
    for (int b = 0; b < nblk; ++b) {
      std::sort(halo[l][b].begin(), halo[l][b].end());
      halo[l][b].erase(std::unique(halo[l][b].begin(), halo[l][b].end()), halo[l][b].end());
    }
  }
  int caph[3] = {0, 0, 0};
  for (int l = 0; l < 3; ++l)
    for (int b = 0; b < nblk; ++b) caph[l] = std::max(caph[l], (int)halo[l][b].size());
  const int cap[3] = {amax * 512, amax * 64, amax * 8};
  if (cap[0] + caph[0] + 1 > 65535) return 0;
  auto local_of = [&](int l, int b, int32_t gslot) -> int32_t {  // own slot or own count + halo position
    const int64_t base = (int64_t)a3ptr[b] << shift[l];
    const int nown = (a3ptr[b + 1] - a3ptr[b]) << shift[l];
    if (owner3[gslot >> shift[l]] == b) return (int32_t)(gslot - base);
    const auto &H = halo[l][b];
    const auto itp = std::lower_bound(H.begin(), H.end(), gslot);
    if (itp == H.end() || *itp != gslot) return -1;
    return nown + (int32_t)(itp - H.begin());
  };
  std::vector<uint16_t> nbr_h[3], cnt_h[3];
  std::vector<double> dinv_h[3], diag_h[3];
  std::vector<int32_t> cell0(nslot[0], -1);
  for (int l = 0; l < 3; ++l) {
    const Lat &F = lat[l];
    nbr_h[l].assign((size_t)6 * nslot[l], 0); cnt_h[l].assign((size_t)6 * nslot[l], 0);
    dinv_h[l].assign(nslot[l], 0.0); diag_h[l].assign(nslot[l], 1.0);
    // empty slots: isolated, every face points at the slot itself (levels 1, 2) or at the zero slot (level 0)
    for (int64_t sl = 0; sl < nslot[l]; ++sl) {
      const int b = owner3[sl >> shift[l]];
      const int nown = (a3ptr[b + 1] - a3ptr[b]) << shift[l];
      const int32_t self = (int32_t)(sl - ((int64_t)a3ptr[b] << shift[l]));
      for (int f = 0; f < 6; ++f) nbr_h[l][(size_t)f * nslot[l] + sl] = (uint16_t)(l == 0 ? nown + (int)halo[0][b].size() : self);
    }
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          if (!F.act[p]) continue;
          const int32_t sl = slot_of(l, p);
          const int b = owner3[sl >> shift[l]];
          double diag = F.dir[p];
          for (int f = 0; f < 6; ++f) {
            diag += (double)F.cnt[f][p] * cfu[f];
            if (F.cnt[f][p] == 0) continue;
            const int32_t loc = local_of(l, b, slot_of(l, F.at(i + dx[f], j + dy[f], k + dz[f])));
            if (loc < 0 || loc > 65535) return 0;
            nbr_h[l][(size_t)f * nslot[l] + sl] = (uint16_t)loc;
            cnt_h[l][(size_t)f * nslot[l] + sl] = (uint16_t)F.cnt[f][p];
          }
          if (!(diag > 0.0)) return 0;
          diag_h[l][sl] = diag;
          dinv_h[l][sl] = omega / diag;
          if (l == 0) cell0[sl] = F.id[p];
        }
  }
  // halo tables: published slot, parent in the next level's local vector
  std::vector<int32_t> hptr[3], hidx[3], hpar[3];
  for (int l = 0; l < 3; ++l) {
    hptr[l].assign(nblk + 1, 0);
    for (int b = 0; b < nblk; ++b) {
      for (int32_t gs : halo[l][b]) {
        hidx[l].push_back(gs);
        int32_t par;
        if (l == 2) par = gs >> 3;                       // global level-3 unknown
        else par = local_of(l + 1, b, gs >> 3);
        if (par < 0) return 0;                           // cannot happen: a fine face implies the coarse face
        hpar[l].push_back(par);
      }
      hptr[l][b + 1] = (int32_t)hidx[l].size();
    }
  }

  // ---- levels 3.. --------------------------------------------------------------------------------------------------------------------------------
  std::vector<int32_t> off_l(nlev, 0);
  int ntot = 0;
  for (int l = 3; l < nlev; ++l) { off_l[l] = ntot; ntot += n_l[l]; }
  std::vector<uint16_t> gnbr((size_t)6 * ntot, 0), gcnt((size_t)6 * ntot, 0), gchild((size_t)8 * ntot, 0xffffu), gpar(ntot, 0);
  std::vector<double> gdinv(ntot, 0.0), gdiag(ntot, 1.0);
  for (int l = 3; l < nlev; ++l) {
    const Lat &F = lat[l];
    for (int k = 0; k < F.d[2]; ++k)
      for (int j = 0; j < F.d[1]; ++j)
        for (int i = 0; i < F.d[0]; ++i) {
          const size_t p = F.at(i, j, k);
          if (!F.act[p]) continue;
          const int me = F.id[p], o = off_l[l] + me;
          double diag = F.dir[p];
          for (int f = 0; f < 6; ++f) {
            diag += (double)F.cnt[f][p] * cfu[f];
            gnbr[(size_t)f * ntot + o] = (uint16_t)me;
            if (F.cnt[f][p] == 0) continue;
            gnbr[(size_t)f * ntot + o] = (uint16_t)F.id[F.at(i + dx[f], j + dy[f], k + dz[f])];
            gcnt[(size_t)f * ntot + o] = (uint16_t)F.cnt[f][p];
          }
          if (!(diag > 0.0)) return 0;
          gdiag[o] = diag;
          gdinv[o] = omega / diag;
          if (l + 1 < nlev) {
            const Lat &P = lat[l + 1];
            const int pid = P.id[P.at(i >> 1, j >> 1, k >> 1)];
            gpar[o] = (uint16_t)pid;
            gchild[(size_t)(((k & 1) << 2) | ((j & 1) << 1) | (i & 1)) * ntot + off_l[l + 1] + pid] = (uint16_t)me;
          }
        }
  }
  std::vector<double> ginv((size_t)nc * nc, 0.0);
  {
    const int o = off_l[nlev - 1];
    for (int i = 0; i < nc; ++i) {
      ginv[(size_t)i * nc + i] += gdiag[o + i];
      for (int f = 0; f < 6; ++f)
        if (gcnt[(size_t)f * ntot + o + i]) ginv[(size_t)i * nc + gnbr[(size_t)f * ntot + o + i]] -= (double)gcnt[(size_t)f * ntot + o + i] * cfu[f];
    }
    if (!dense_inverse(ginv, nc)) return 0;
  }

  // ---- shared memory, upload ------------------------------------------------------------------------------------------------------------------------
  auto pad_d = [](size_t n) { return ((n + 1) & ~(size_t)1) * 8; };
  auto pad_h = [](size_t n) { return ((n + 7) & ~(size_t)7) * 2; };
  auto pad_i = [](size_t n) { return ((n + 3) & ~(size_t)3) * 4; };
  size_t smem = 3 * pad_d(cap[0]) + pad_d(cap[0] + caph[0] + 2);
  for (int l = 1; l < 3; ++l) smem += pad_d(cap[l] + caph[l] + 2) + 5 * pad_d(cap[l]) + 2 * pad_h((size_t)6 * cap[l]);
  smem += 6 * pad_d(ntot) + pad_d((size_t)nc * nc) + pad_d(64);
  for (int l = 0; l < 3; ++l) smem += 2 * pad_i(caph[l]);
  smem += 2 * pad_h((size_t)6 * ntot) + pad_h((size_t)8 * ntot) + pad_h(ntot);
  if (smem > 225 * 1024) return 0;

  MgPlan *P = new MgPlan();
  MgArgs &a = P->a;
  a.nblk = nblk; a.n_act = na; a.omega = omega; a.tau = tau; a.rho = omega2 / omega;
  for (int f = 0; f < 6; ++f) a.cfu[f] = cfu[f];
  a.a3ptr = A.put(a3ptr);
  for (int l = 0; l < 3; ++l) {
    a.hptr[l] = A.put(hptr[l]);
    if (hidx[l].empty()) { hidx[l].push_back(0); hpar[l].push_back(0); }
    a.hidx[l] = A.put(hidx[l]); a.hpar[l] = A.put(hpar[l]);
  }
  {  // everything that crosses CTA borders in one block (zeroed before every launch)
    size_t nd = 0;
    for (int l = 0; l < 3; ++l) nd += (size_t)4 * nslot[l];
    nd += (size_t)2 * n3 + (size_t)8 * nblk + 64;
    double *blk = A.zeros<double>(nd);
    a.xbuf = blk; a.xbuf_bytes = nd * sizeof(double);
    for (int l = 0; l < 3; ++l) { a.xg[l] = blk; blk += (size_t)2 * nslot[l]; a.xu[l] = blk; blk += (size_t)2 * nslot[l]; }
    a.g3 = blk; blk += (size_t)2 * n3;
    a.part = blk;
  }
  a.cell0 = A.put(cell0); a.nbr0 = A.put(nbr_h[0]); a.dinv0 = A.put(dinv_h[0]); a.diag0 = A.put(diag_h[0]);
  for (int l = 1; l < 3; ++l) { a.nbr[l] = A.put(nbr_h[l]); a.cnt[l] = A.put(cnt_h[l]); a.dinv[l] = A.put(dinv_h[l]); a.diag[l] = A.put(diag_h[l]); }
  a.nbr[0] = nullptr; a.cnt[0] = nullptr; a.dinv[0] = nullptr; a.diag[0] = nullptr;
  a.nlev = nlev; a.ntot = ntot;
  for (int l = 0; l < kMgMaxLevels; ++l) { a.n_l[l] = l < nlev ? n_l[l] : 0; a.off_l[l] = l < nlev ? off_l[l] : 0; }
  a.gnbr = A.put(gnbr); a.gcnt = A.put(gcnt); a.gchild = A.put(gchild); a.gpar = A.put(gpar);
  a.gdinv = A.put(gdinv); a.gdiag = A.put(gdiag); a.ginv = A.put(ginv);
  a.xprev = A.zeros<double>((size_t)2 * nslot[0]);
  a.gpart = A.zeros<double>((size_t)8 * nblk + 8);
  a.bar = A.zeros<unsigned int>(4);
  a.cap0 = cap[0]; a.caph0 = caph[0]; a.cap1 = cap[1]; a.caph1 = caph[1]; a.cap2 = cap[2]; a.caph2 = caph[2];
  P->cpt = cpt; P->smem = smem; P->levels = nlev;
  if (A.rc < 0) { delete P; return A.rc; }
  h->mg = P;
  return 0;
}

int nb_mg_solve(nanobte_solver *h) {
  MgPlan &P = *h->mg;
  MgArgs a = P.a;
  a.max_iter = h->cg_max_iter; a.B = h->B; a.rtol = h->cg_rtol; a.beta = h->beta;
  a.vol = h->vol; a.theta_SI = h->theta_SI; a.theta_prev = h->theta_prev; a.faceflux = h->bd.faceflux; a.bf_area = h->bd.bf_area;
  a.rhs_direct = h->cg_rhs_direct;
  // the band sum of the face fluxes (R14c') once per face by a small kernel, in band order as the in-kernel loop would add
  // them: 30 strided loads per wall face are 15 us of the solve when the cooperative kernel does them itself
  if (!h->leak_imported && !a.rhs_direct && h->n_bf > 0) {
    int rc = nb_launch_leak_sum(h);
    if (rc < 0) return rc;
  }
  a.leak_sum = (h->leak_imported || (!a.rhs_direct && h->n_bf > 0)) ? h->leak_sum : nullptr;
  a.nprev = h->cgf_nprev;  // the history counter of the handle (reset by solve / set_T / a failed or foreign solve)
  h->cgf_nprev = std::min(2, h->cgf_nprev + 1);
  a.cellbf_ptr = h->cellbf_ptr; a.cellbf = h->cellbf; a.x = h->cg_x; a.iters_out = h->d_maxdT + 1;
  mg_fn fn = mg_pick(P.cpt);
  if (!fn) return nb_fail(h, NANOBTE_E_INVALID, "internal: no multigrid CG variant for %d slots per thread", P.cpt);
  NB_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P.smem));
  NB_CUDA(h, cudaMemsetAsync(a.bar, 0, sizeof(unsigned int), h->stream));
  NB_CUDA(h, cudaMemsetAsync(a.xbuf, 0, a.xbuf_bytes, h->stream));  // sequence bits start from zero (see mg_tag)
  void *args[] = {&a};
  NB_CUDA(h, cudaLaunchCooperativeKernel((void *)fn, dim3(a.nblk), dim3(kMgThreads), args, P.smem, h->stream));
  h->launches++;
  return 0;
}

#ifdef MG_PROF
extern "C" int nanobte_debug_mg_prof(unsigned long long *out, int reset) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(out, g_mg_prof, sizeof(unsigned long long) * 16);
  if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(g_mg_prof, z, sizeof(z)); }
  return 0;
}
#endif

void nb_free_mg(nanobte_solver *h) {
  delete h->mg;
  h->mg = nullptr;
}
