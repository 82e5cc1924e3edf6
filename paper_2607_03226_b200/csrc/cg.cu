// cg.cu -- (a7) synthetic correction: right-hand side and an unpreconditioned conjugate gradient on the
// two-point-flux finite-volume diffusion operator (Eq. 8-12; readings R14a-e), as ONE persistent
// cooperative kernel: two grid barriers per CG iteration, all scalars on the device, no host synchronisation
// inside the loop.  Reductions use a fixed tree (block partials summed in block order by every block), so the
// result is bitwise reproducible and identical in every block.
//
//   A delta = rhs,  (A x)_c = sum_{f interior} kappa A_f (x_c - x_N(c,f))/d_f + sum_{f thermalizing} kappa A_f x_c/d_cf
//   rhs_c   = V_c beta (theta_SI,c - theta^n_c) + sum_{f reflecting of c} A_f F_f          (R14c, R14c')
//   CG from delta = 0, stop at ||r||^2 <= rtol^2 ||rhs||^2                               (R14e)
#include <cooperative_groups.h>

#include "cg_mg.h"
#include "internal.h"
namespace cg = cooperative_groups;

// bit set in the iteration count the kernels report when the loop ended on max_iter with ||r|| > rtol ||rhs||
constexpr unsigned long long kCgNotConverged = 1ull << 40;

struct CgArgs {
  int32_t n, nf, max_iter, B;
  const int32_t *nbr;    // [nf][n]  neighbour (active index); entries without a neighbour point at the cell itself
  const double *coef;    // [nf][n]  kappa A_f / d_f for interior faces, 0 otherwise
  const double *diag;    // [n]      sum of interior + thermalizing face coefficients
  const double *vol, *theta_SI, *theta_prev, *faceflux, *bf_area;
  const double *rhs_direct;  // non-null: the right-hand side itself (Fourier initial guess, R21)
  const double *leak_sum;    // non-null: [n_bf] the face leak summed over all bands (band shards)
  const int32_t *cellbf_ptr, *cellbf;
  double *x, *r, *p0, *p1, *ap, *partial;
  unsigned long long *iters_out;
  double beta, rtol;
};

__device__ __forceinline__ double block_sum(double v, double *red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x < 32) {
    s = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  }
  __syncthreads();
  return s;  // valid in warp 0
}

// every block sums the per-block partials in the same order -> identical value everywhere
__device__ __forceinline__ double grid_total(const double *partial, int nblk, double *red) {
  double s = 0.0;
  if (threadIdx.x < 32) {
    for (int k = threadIdx.x; k < nblk; k += 32) s += __ldcg(partial + k);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) red[32] = s;
  }
  __syncthreads();
  s = red[32];
  __syncthreads();
  return s;
}

__global__ void __launch_bounds__(256) cg_kernel(CgArgs a) {
  __shared__ double red[40];
  cg::grid_group grid = cg::this_grid();
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x, nblk = gridDim.x;
  // right-hand side, x = 0, r = rhs, p_old = rhs
  double loc = 0.0;
  for (int i = tid; i < a.n; i += nth) {
    double rhs;
    if (a.rhs_direct) {
      rhs = a.rhs_direct[i];
    } else {
      rhs = a.vol[i] * a.beta * (a.theta_SI[i] - a.theta_prev[i]);
      for (int k = a.cellbf_ptr[i]; k < a.cellbf_ptr[i + 1]; ++k) {
        const int bf = a.cellbf[k];
        double F = 0.0;
        if (a.leak_sum) F = a.leak_sum[bf];
        else for (int b = 0; b < a.B; ++b) F += a.faceflux[(size_t)bf * a.B + b];
        rhs += a.bf_area[bf] * F;
      }
    }
    a.x[i] = 0.0;
    a.r[i] = rhs;
    a.p0[i] = rhs;
    loc += rhs * rhs;
  }
  loc = block_sum(loc, red);
  if (threadIdx.x == 0) a.partial[blockIdx.x] = loc;
  grid.sync();
  const double bb = grid_total(a.partial, nblk, red);
  const double stop2 = a.rtol * a.rtol * bb;
  double rr = bb, bet = 0.0;
  double *pold = a.p0, *pnew = a.p1;
  double *part_a = a.partial + 2048, *part_b = a.partial;  // alternate so a slow block never reads a recycled slot
  int it = 0;
  while (rr > stop2 && it < a.max_iter) {
    // p_new = r + bet p_old (own entry stored, neighbours' recomputed), Ap, p.Ap
    loc = 0.0;
    for (int i = tid; i < a.n; i += nth) {
      const double pi = a.r[i] + bet * pold[i];
      double acc = a.diag[i] * pi;
      for (int f = 0; f < a.nf; ++f) {
        const int j = a.nbr[(size_t)f * a.n + i];
        acc -= a.coef[(size_t)f * a.n + i] * (a.r[j] + bet * pold[j]);
      }
      pnew[i] = pi;
      a.ap[i] = acc;
      loc += pi * acc;
    }
    loc = block_sum(loc, red);
    if (threadIdx.x == 0) part_a[blockIdx.x] = loc;
    grid.sync();
    const double pAp = grid_total(part_a, nblk, red);
    const double alpha = rr / pAp;
    loc = 0.0;
    for (int i = tid; i < a.n; i += nth) {
      a.x[i] += alpha * pnew[i];
      const double ri = a.r[i] - alpha * a.ap[i];
      a.r[i] = ri;
      loc += ri * ri;
    }
    loc = block_sum(loc, red);
    if (threadIdx.x == 0) part_b[blockIdx.x] = loc;
    grid.sync();
    const double rr_new = grid_total(part_b, nblk, red);
    bet = rr_new / rr;
    rr = rr_new;
    double *t = pold; pold = pnew; pnew = t;
    ++it;
  }
  if (tid == 0) *a.iters_out = (unsigned long long)it | (rr > stop2 ? kCgNotConverged : 0ull);
}

// =================================================================================================================
// Fused variant (the one used whenever the plan built at create fits): one CTA per contiguous chunk of cells, the
// CTA's slice of every CG vector in registers, the residual of the chunk plus its halo in shared memory, and ONE
// grid barrier per iteration.
//   * Single-reduction CG (Chronopoulos & Gear): with s = A p and w = A r kept by recurrence,
//       beta = g_k / g_{k-1},  alpha = g_k / (d_k - beta g_k / alpha_{k-1}),  g = (r, r),  d = (w, r),
//       p <- r + beta p,  s <- w + beta s,  x <- x + alpha p,  r <- r - alpha s,  w <- A r
//     so both dot products of an iteration are reduced together.  Same iterates as textbook CG in exact arithmetic.
//   * No halo exchange of r: a CTA applies the same two recurrences (s, r) to its halo cells, redundantly and with
//     bit-identical arithmetic, reading only the owner's published w.  Hence the barrier that completes the
//     reduction is the only grid-wide synchronisation of an iteration.
//   * Reductions are fixed trees (per-CTA partials summed in CTA order by every warp): bitwise reproducible and
//     identical in every CTA, which is what keeps the redundant halo copies consistent.
// =================================================================================================================
struct CgfArgs {
  int32_t n, nf, nblk, chunk, nh_cap, max_iter, B;
  const int32_t *nloc, *perm;
  const double *coef, *diag, *vol, *theta_SI, *theta_prev, *faceflux, *bf_area;
  const double *rhs_direct;  // non-null: the right-hand side itself (Fourier initial guess, R21)
  const double *leak_sum;    // non-null: [n_bf] the face leak summed over all bands (band shards)
  const int32_t *cellbf_ptr, *cellbf, *hptr, *hidx;
  double *x, *w, *part;
  unsigned int *bar;
  unsigned long long *iters_out;
  double beta, rtol;
  double cfu[6];  // face-uniform stencil: the one non-zero coefficient of every face slot
  // recycled initial guess: the last (up to) two solutions, in CG order, and a reduction buffer
  int32_t nprev;
  double *xprev;    // [2][n]
  double *gpart;    // [nblk][8]
};

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

constexpr int kCgfThreads = 512;

// UNI: every face slot carries one coefficient value or none (uniform structured grids).  The coefficients are then
// kernel parameters, and a missing neighbour points at a slot of r_loc that stays zero.
template <int NF, int CPT, bool UNI>
__global__ void __launch_bounds__(kCgfThreads, 1) cg_fused_kernel(CgfArgs a) {
  extern __shared__ __align__(16) unsigned char cgf_smem[];
  double *r_loc = reinterpret_cast<double *>(cgf_smem);           // [chunk + nh_cap]
  double *s_h = r_loc + a.chunk + a.nh_cap;                       // [nh_cap]
  double *x_s = s_h + a.nh_cap;                                   // [chunk]  solution (kept out of the registers)
  double *p_s = x_s + a.chunk;                                    // [chunk]  search direction
  int32_t *hidx_s = reinterpret_cast<int32_t *>(p_s + a.chunk);   // [nh_cap]
  __shared__ double red[2 * (kCgfThreads / 32)];
  __shared__ double gd[2];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int k = blockIdx.x, a0 = k * a.chunk, nown = min(a.n, a0 + a.chunk) - a0;
  const int h0 = a.hptr[k], nh = a.hptr[k + 1] - h0;
  const int n = a.n;
  for (int j = tid; j < nh; j += kCgfThreads) {
    hidx_s[j] = a.hidx[h0 + j];
    s_h[j] = 0.0;
  }
  if (tid == 0) r_loc[a.chunk + a.nh_cap - 1] = 0.0;  // the last halo slot belongs to no CTA's halo: the zero slot
  // Stencil of the thread's cells: in registers up to 2 cells per thread; with 4 the 48 coefficient registers would
  // spill, so the coefficients are re-read every iteration through the read-only path (95 KB per CTA: L1-resident).
  constexpr bool kStencilInRegs = CPT <= 2 && !UNI;
  constexpr int CR = kStencilInRegs ? CPT : 1;
  double cf[CR][NF], dg[CPT], r[CPT], s[CPT], wv[CPT];
  uint16_t nl[CPT][NF];  // local indices < 65536 (checked when the plan is built); always in registers
#pragma unroll
  for (int c = 0; c < CPT; ++c) {
    const int li = tid + c * kCgfThreads, i = a0 + li;
    s[c] = wv[c] = r[c] = dg[c] = 0.0;
    if (li < a.chunk) x_s[li] = p_s[li] = 0.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      nl[c][f] = 0;
      if (kStencilInRegs) cf[c % CR][f] = 0.0;
    }
    if (li < nown) {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        nl[c][f] = (uint16_t)a.nloc[(size_t)f * n + i];
        if (kStencilInRegs) cf[c % CR][f] = a.coef[(size_t)f * n + i];
      }
      dg[c] = a.diag[i];
      const int io = a.perm[i];  // the cell in the solver's own (active) numbering
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
      r_loc[li] = rhs;
      a.w[(size_t)n + i] = rhs;  // publish r_0 through the second w buffer
    }
  }
  unsigned int epoch = 1;
  // ---- recycled initial guess ---------------------------------------------------------------------------------------
  // The operator never changes and, as the outer iteration settles on its slowest mode, successive corrections become
  // collinear: x_0 = Galerkin projection of the new right-hand side on the span of the last two solutions X1, X2
  // (2 x 2 system with X_i^T A X_j and X_i^T b) starts the CG with a residual orders of magnitude below ||b||.  The
  // stopping rule is unchanged (||r|| <= rtol ||b||).  X1, X2 were written by the previous launches, so their halo
  // values are simply read; the only communication is one reduction of six scalars.
  double bb_total = -1.0;  // < 0: not computed (no history): ||b||^2 is then the first gamma
  if (a.nprev > 0) {
    double X[2][CPT], AX[2][CPT];
#pragma unroll
    for (int v = 0; v < 2; ++v) {
      const double *xv = a.xprev + (size_t)v * n;
      const bool have = v < a.nprev;
      __syncthreads();  // r_loc is reused as the scratch vector of each pass
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const int li = tid + c * kCgfThreads;
        X[v][c] = (have && li < nown) ? xv[a0 + li] : 0.0;
        if (li < nown) r_loc[li] = X[v][c];
      }
      for (int j = tid; j < nh; j += kCgfThreads) r_loc[a.chunk + j] = have ? xv[hidx_s[j]] : 0.0;
      __syncthreads();
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const int li = tid + c * kCgfThreads;
        AX[v][c] = 0.0;
        if (li < nown) {
          double acc = dg[c] * X[v][c];
#pragma unroll
          for (int f = 0; f < NF; ++f) {
            if (UNI) acc -= a.cfu[f] * r_loc[nl[c][f]];
            else if (kStencilInRegs) acc -= cf[c % CR][f] * r_loc[nl[c][f]];
            else acc -= __ldg(a.coef + (size_t)f * n + a0 + li) * r_loc[nl[c][f]];
          }
          AX[v][c] = acc;
        }
      }
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
    __shared__ double red6[6 * (kCgfThreads / 32)];
#pragma unroll
    for (int q = 0; q < 6; ++q) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sums[q] += __shfl_xor_sync(0xffffffffu, sums[q], o);
      if (lane == 0) red6[q * (kCgfThreads / 32) + wid] = sums[q];
    }
    __syncthreads();
    if (tid < 6) {
      double t = 0.0;
      for (int w2 = 0; w2 < kCgfThreads / 32; ++w2) t += red6[tid * (kCgfThreads / 32) + w2];
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
      const int li = tid + c * kCgfThreads;
      if (li < nown) {
        x_s[li] = c1 * X[0][c] + c2 * X[1][c];
        r[c] -= c1 * AX[0][c] + c2 * AX[1][c];
        r_loc[li] = r[c];
        a.w[(size_t)n + a0 + li] = r[c];
      }
    }
  }
  grid_barrier(a.bar, epoch++ * a.nblk);
  for (int j = tid; j < nh; j += kCgfThreads) r_loc[a.chunk + j] = __ldcg(a.w + (size_t)n + hidx_s[j]);
  __syncthreads();

  // w = A r on the chunk, the two partial dot products, publication of w; reads r_loc
  auto apply_and_reduce = [&](int par_out) {
    double g = 0.0, d = 0.0;
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kCgfThreads;
      if (li < nown) {
        double acc = dg[c] * r[c];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          if (UNI) acc -= a.cfu[f] * r_loc[nl[c][f]];
          else if (kStencilInRegs) acc -= cf[c % CR][f] * r_loc[nl[c][f]];
          else acc -= __ldg(a.coef + (size_t)f * n + a0 + li) * r_loc[nl[c][f]];
        }
        wv[c] = acc;
        a.w[(size_t)par_out * n + a0 + li] = acc;
        g += r[c] * r[c];
        d += acc * r[c];
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      g += __shfl_xor_sync(0xffffffffu, g, o);
      d += __shfl_xor_sync(0xffffffffu, d, o);
    }
    if (lane == 0) { red[2 * wid] = g; red[2 * wid + 1] = d; }
    __syncthreads();
    if (wid == 0) {
      double G = lane < kCgfThreads / 32 ? red[2 * lane] : 0.0, D = lane < kCgfThreads / 32 ? red[2 * lane + 1] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        G += __shfl_xor_sync(0xffffffffu, G, o);
        D += __shfl_xor_sync(0xffffffffu, D, o);
      }
      if (lane == 0) *reinterpret_cast<double2 *>(a.part + ((size_t)par_out * a.nblk + k) * 2) = make_double2(G, D);
    }
  };
  apply_and_reduce(0);
  grid_barrier(a.bar, epoch++ * a.nblk);

  double g_prev = 1.0, alpha_prev = 1.0, stop2 = 0.0;
  int it = 0;
  bool not_converged = false;
  for (;; ++it) {
    const int par = it & 1;
    // Issue every global load of the iteration first (per-CTA partials and the owners' w of the first halo batch):
    // one L2 round trip after the barrier instead of two.
    const double *pp = a.part + (size_t)par * a.nblk * 2;
    const double *wp = a.w + (size_t)par * n;
    constexpr int NP = 5, HB = 10;
    double2 pv[NP];
    if (wid == 0) {  // one warp per CTA reads the partials: 2368 warps hammering the same 19 lines is an L2 hot spot
#pragma unroll
      for (int u = 0; u < NP; ++u) {
        const int q = lane + 32 * u;
        pv[u] = q < a.nblk ? __ldcg(reinterpret_cast<const double2 *>(pp) + q) : make_double2(0.0, 0.0);
      }
    }
    double wh[HB];
#pragma unroll
    for (int q = 0; q < HB; ++q) {
      const int j = tid + q * kCgfThreads;
      wh[q] = j < nh ? __ldcg(wp + hidx_s[j]) : 0.0;
    }
    // fixed summation order -> the same bits in every CTA
    if (wid == 0) {
      double g = 0.0, d = 0.0;
#pragma unroll
      for (int u = 0; u < NP; ++u) {
        g += pv[u].x;
        d += pv[u].y;
      }
      for (int q = lane + 32 * NP; q < a.nblk; q += 32) {  // more than 160 CTAs: not on B200
        const double2 v = __ldcg(reinterpret_cast<const double2 *>(pp) + q);
        g += v.x;
        d += v.y;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        g += __shfl_xor_sync(0xffffffffu, g, o);
        d += __shfl_xor_sync(0xffffffffu, d, o);
      }
      if (lane == 0) { gd[0] = g; gd[1] = d; }
    }
    __syncthreads();
    const double g = gd[0], d = gd[1];
    if (it == 0) stop2 = a.rtol * a.rtol * (bb_total >= 0.0 ? bb_total : g);
    if (!(g > stop2)) break;
    if (it >= a.max_iter) { not_converged = true; break; }
    const double bet = it ? g / g_prev : 0.0;
    const double alpha = it ? g / (d - bet * g / alpha_prev) : g / d;
    // halo copies: same recurrences as the owner, owner's w
#pragma unroll
    for (int q = 0; q < HB; ++q) {
      const int j = tid + q * kCgfThreads;
      if (j < nh) {
        const double sh = fma(bet, s_h[j], wh[q]);
        s_h[j] = sh;
        r_loc[a.chunk + j] = fma(-alpha, sh, r_loc[a.chunk + j]);
      }
    }
    for (int j = tid + HB * kCgfThreads; j < nh; j += kCgfThreads) {  // very large halos: one more round trip each
      const double sh = fma(bet, s_h[j], __ldcg(wp + hidx_s[j]));
      s_h[j] = sh;
      r_loc[a.chunk + j] = fma(-alpha, sh, r_loc[a.chunk + j]);
    }
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int li = tid + c * kCgfThreads;
      if (li < nown) {
        const double pc = fma(bet, p_s[li], r[c]);
        p_s[li] = pc;
        s[c] = fma(bet, s[c], wv[c]);
        x_s[li] = fma(alpha, pc, x_s[li]);
        r[c] = fma(-alpha, s[c], r[c]);
        r_loc[li] = r[c];
      }
    }
    __syncthreads();
    apply_and_reduce(par ^ 1);
    grid_barrier(a.bar, epoch++ * a.nblk);
    g_prev = g;
    alpha_prev = alpha;
  }
#pragma unroll
  for (int c = 0; c < CPT; ++c) {
    const int li = tid + c * kCgfThreads;
    if (li < nown) {
      a.x[a.perm[a0 + li]] = x_s[li];
      a.xprev[(size_t)n + a0 + li] = a.xprev[a0 + li];  // history of the recycled initial guess
      a.xprev[a0 + li] = x_s[li];
    }
  }
  if (k == 0 && tid == 0) *a.iters_out = (unsigned long long)it | (not_converged ? kCgNotConverged : 0ull);
}

typedef void (*cgf_fn)(CgfArgs);
template <int NF, bool UNI>
static cgf_fn cgf_pick_cpt(int cpt) {
  switch (cpt) {
    case 1: return cg_fused_kernel<NF, 1, UNI>;
    case 2: return cg_fused_kernel<NF, 2, UNI>;
    case 4: return cg_fused_kernel<NF, 4, UNI>;
    case 8: return cg_fused_kernel<NF, 8, UNI>;
  }
  return nullptr;
}
static cgf_fn cgf_pick(int nf, int cpt, bool uni) {
  switch (nf) {
    case 3: return uni ? cgf_pick_cpt<3, true>(cpt) : cgf_pick_cpt<3, false>(cpt);
    case 4: return uni ? cgf_pick_cpt<4, true>(cpt) : cgf_pick_cpt<4, false>(cpt);
    case 6: return uni ? cgf_pick_cpt<6, true>(cpt) : cgf_pick_cpt<6, false>(cpt);
  }
  return nullptr;
}

static int cg_solve_fused(nanobte_solver *h) {
  cgf_fn fn = cgf_pick(h->cg_nf, h->cgf_cpt, h->cgf_uni);
  if (!fn) return nb_fail(h, NANOBTE_E_INVALID, "internal: no fused CG variant for nf=%d cpt=%d", h->cg_nf, h->cgf_cpt);
  CgfArgs a;
  a.n = h->n_act; a.nf = h->cg_nf; a.nblk = h->cgf_nblk; a.chunk = h->cgf_chunk; a.nh_cap = h->cgf_nh_cap;
  a.max_iter = h->cg_max_iter; a.B = h->B;
  a.nloc = h->cgf_nloc; a.perm = h->cgf_perm; a.coef = h->cgf_coef; a.diag = h->cgf_diag; a.vol = h->vol;
  a.theta_SI = h->theta_SI; a.theta_prev = h->theta_prev; a.faceflux = h->bd.faceflux; a.bf_area = h->bd.bf_area;
  a.cellbf_ptr = h->cellbf_ptr; a.cellbf = h->cellbf; a.hptr = h->cgf_hptr; a.hidx = h->cgf_hidx;
  a.rhs_direct = h->cg_rhs_direct;
  a.leak_sum = h->leak_imported ? h->leak_sum : nullptr;
  a.x = h->cg_x; a.w = h->cgf_w; a.part = h->cgf_part; a.bar = h->cgf_bar;
  a.iters_out = h->d_maxdT + 1;
  a.beta = h->beta; a.rtol = h->cg_rtol;
  for (int f = 0; f < 6; ++f) a.cfu[f] = h->cgf_cfu[f];
  a.nprev = h->cgf_recycle ? h->cgf_nprev : 0; a.xprev = h->cgf_xprev; a.gpart = h->cgf_gpart;
  h->cgf_nprev = std::min(2, h->cgf_nprev + 1);
  NB_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->cgf_smem));
  NB_CUDA(h, cudaMemsetAsync(h->cgf_bar, 0, sizeof(unsigned int), h->stream));
  void *args[] = {&a};
  NB_CUDA(h, cudaLaunchCooperativeKernel((void *)fn, dim3(h->cgf_nblk), dim3(kCgfThreads), args, h->cgf_smem, h->stream));
  h->launches++;
  return 0;
}

int nb_cg_blocks(nanobte_solver *h) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cg_kernel, 256, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  int want = (h->n_act + 255) / 256;
  int cap = std::min(per_sm * h->n_sm, 2048);
  return std::max(1, std::min(want, cap));
}

int nb_cg_solve(nanobte_solver *h, int *iters) {
  if (iters) *iters = -1;  // read back by the caller together with max|dT|
  if (h->mg && !h->cg_force_generic) return nb_mg_solve(h);
  if (h->cgf_ok && !h->cg_force_generic) return cg_solve_fused(h);
  CgArgs a;
  a.n = h->n_act; a.nf = h->cg_nf; a.max_iter = h->cg_max_iter; a.B = h->B;
  a.nbr = h->cg_nbr; a.coef = h->cg_coef; a.diag = h->cg_diag;
  a.vol = h->vol; a.theta_SI = h->theta_SI; a.theta_prev = h->theta_prev;
  a.faceflux = h->bd.faceflux; a.bf_area = h->bd.bf_area; a.cellbf_ptr = h->cellbf_ptr; a.cellbf = h->cellbf;
  a.rhs_direct = h->cg_rhs_direct;
  a.leak_sum = h->leak_imported ? h->leak_sum : nullptr;
  a.x = h->cg_x; a.r = h->cg_r; a.p0 = h->cg_p0; a.p1 = h->cg_p1; a.ap = h->cg_rhs; a.partial = h->cg_partial;
  a.iters_out = h->d_maxdT + 1;
  a.beta = h->beta; a.rtol = h->cg_rtol;
  if (h->cg_blocks == 0) h->cg_blocks = nb_cg_blocks(h);
  void *args[] = {&a};
  NB_CUDA(h, cudaLaunchCooperativeKernel((void *)cg_kernel, dim3(h->cg_blocks), dim3(256), args, 0, h->stream));
  h->launches++;
  if (iters) *iters = -1;  // read back by the caller together with max|dT|
  return 0;
}
