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

#include "internal.h"
namespace cg = cooperative_groups;

struct CgArgs {
  int32_t n, nf, max_iter, B;
  const int32_t *nbr;    // [nf][n]  neighbour (active index); entries without a neighbour point at the cell itself
  const double *coef;    // [nf][n]  kappa A_f / d_f for interior faces, 0 otherwise
  const double *diag;    // [n]      sum of interior + thermalizing face coefficients
  const double *vol, *theta_SI, *theta_prev, *faceflux, *bf_area;
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
    double rhs = a.vol[i] * a.beta * (a.theta_SI[i] - a.theta_prev[i]);
    for (int k = a.cellbf_ptr[i]; k < a.cellbf_ptr[i + 1]; ++k) {
      const int bf = a.cellbf[k];
      double F = 0.0;
      for (int b = 0; b < a.B; ++b) F += a.faceflux[(size_t)bf * a.B + b];
      rhs += a.bf_area[bf] * F;
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
  if (tid == 0) *a.iters_out = (unsigned long long)it;
}

int nb_cg_blocks(nanobte_solver *h) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cg_kernel, 256, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  int want = (h->n_act + 255) / 256;
  int cap = std::min(per_sm * h->n_sm, 2048);
  return std::max(1, std::min(want, cap));
}

int nb_cg_solve(nanobte_solver *h, int *iters) {
  CgArgs a;
  a.n = h->n_act; a.nf = h->cg_nf; a.max_iter = h->cg_max_iter; a.B = h->B;
  a.nbr = h->cg_nbr; a.coef = h->cg_coef; a.diag = h->cg_diag;
  a.vol = h->vol; a.theta_SI = h->theta_SI; a.theta_prev = h->theta_prev;
  a.faceflux = h->bd.faceflux; a.bf_area = h->bd.bf_area; a.cellbf_ptr = h->cellbf_ptr; a.cellbf = h->cellbf;
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
