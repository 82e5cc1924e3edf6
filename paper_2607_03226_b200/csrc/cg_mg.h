// cg_mg.h -- private declarations of the multigrid-preconditioned conjugate gradient for the synthetic correction (a7) on
// uniform 3-D structured grids (cg_mg.cu).  Same linear system and stopping rule as cg.cu (R14a-e: A delta = rhs,
// ||r|| <= rtol ||rhs||); what changes is the iterate sequence -- DESIGN.md section 3, reading R14e'.
#pragma once
#include <cstdint>
#include <vector>

#include "host_util.h"
#include "internal.h"

constexpr int kMgThreads = 512;
constexpr int kMgDist = 3;        // levels 0, 1, 2 are distributed over the CTAs (chunk = whole 8 x 8 x 8 blocks of cells)
constexpr int kMgMaxLevels = 10;  // levels 3.. are small and held by every CTA in shared memory
constexpr int kMgCoarsest = 32;   // the coarsest level is solved with its dense inverse

// Everything the kernel reads, by level.  Slots: a CTA owns na3 level-3 aggregates (8^3 blocks of the cell lattice); its
// level-l slot (l = 0, 1, 2) of aggregate a is a * 8^(3-l) + the octree path below the aggregate, so parent(slot) =
// slot >> 3 and the 8 children of a slot are consecutive.  Slots without a cell (mask, lattice edge) are isolated unknowns
// with a zero right-hand side.
struct MgArgs {
  int32_t nblk, n_act, max_iter, B;
  double rtol, beta, omega, tau;
  double rho;                      // second Jacobi step's damping over the first's (the dinv arrays carry the first's)
  double cfu[6];                   // kappa A_f / d_f of the six face directions (-x +x -y +y -z +z)
  // per CTA: [nblk + 1] prefix offsets
  const int32_t *a3ptr;            // level-3 aggregates (= global level-3 unknowns, CTA-contiguous)
  const int32_t *hptr[kMgDist];    // halo lists of levels 0, 1, 2
  // level 0 (per global slot, 512 per aggregate)
  const int32_t *cell0;            // active-cell index of the slot, -1 = empty slot
  const uint16_t *nbr0;            // [6][nslot0] local index (own slot | own count + halo position | the zero slot)
  const double *dinv0;             // omega / diagonal (empty slot: 0)
  const double *diag0;             // diagonal (empty slot: 1)
  // levels 1, 2 (per global slot)
  const uint16_t *nbr[kMgDist];    // [6][nslot_l] local index (a face without a neighbour: the slot itself, count 0)
  const uint16_t *cnt[kMgDist];    // [6][nslot_l] fine faces behind the coarse face: coefficient = cnt * cfu[f]
  const double *dinv[kMgDist], *diag[kMgDist];
  // halo entries of levels 0, 1, 2: where the value is published, and the entry's parent in the next level's local vector
  // (levels 0, 1: own slot or own count + halo position; level 2: global level-3 unknown)
  const int32_t *hidx[kMgDist];
  const int32_t *hpar[kMgDist];
  // published iterates per global slot, [2][nslot_l] each (double-buffered by iteration parity): xg = on the way down,
  // xu = on the way up (level 0: u).  Every published value carries a sequence bit in its last mantissa bit (see
  // exchange() in cg_mg.cu), so a reader needs no barrier: it re-reads until the bit is the current one.
  double *xg[kMgDist], *xu[kMgDist];
  void *xbuf; size_t xbuf_bytes;   // all of them, g3 and part: zeroed before every launch
  // levels 3 .. nlev-1, the same in every CTA
  int32_t nlev, n_l[kMgMaxLevels], off_l[kMgMaxLevels];  // unknowns per level, offset of the level in the arrays below
  const uint16_t *gnbr, *gcnt;     // [6][ntot]   (index inside the level)
  const uint16_t *gchild;          // [8][ntot]   children in the level below (0xffff: none); level 3: unused
  const uint16_t *gpar;            // [ntot]      parent in the level above
  const double *gdinv, *gdiag;     // [ntot]
  const double *ginv;              // [nc][nc] inverse of the coarsest operator
  double *g3;                      // [2][n3] published level-3 right-hand side (tagged like the iterates)
  // recycled initial guess (as in cg.cu): the last two solutions per level-0 slot, and a reduction buffer
  int32_t nprev;
  double *xprev;                   // [2][nslot0]
  double *gpart;                   // [nblk][8]
  // right-hand side, result, reductions
  const double *vol, *theta_SI, *theta_prev, *faceflux, *bf_area;
  const double *rhs_direct;        // non-null: the right-hand side itself (Fourier initial guess, R21)
  const double *leak_sum;          // non-null: [n_bf] the face leak summed over all bands (band shards)
  const int32_t *cellbf_ptr, *cellbf;
  double *x;                       // [n_act] solution, active-cell order
  double *part;                    // [2][nblk][4] tagged partial dot products
  unsigned int *bar;
  unsigned long long *iters_out;
  // shared-memory carve-up (element counts, the same for every CTA: maxima over the CTAs)
  int32_t cap0, caph0, cap1, caph1, cap2, caph2, ntot;
};

struct MgPlan {
  MgArgs a{};
  int cpt = 0;        // level-0 slots per thread
  size_t smem = 0;
  int levels = 0;
};

int nb_mg_build(nanobte_solver *h, Arena &A, const GenericTables &g, const double *cfu, const int grid[3]);
int nb_mg_solve(nanobte_solver *h);
void nb_free_mg(nanobte_solver *h);
