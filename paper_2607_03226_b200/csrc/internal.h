// internal.h -- private declarations of libnanobte (CUDA, sm_100a).  Not part of the ABI (include/nanobte.h).
//
// Data layout in HBM:
//   e      [D][B][n_pos]         one contiguous row per (direction, band) system, cells in the sweep order of
//                                the direction's class (octant hyperplane order / per-direction level order)
//   bin    per direction d: [B][n_in(class(d))]   boundary inflow values consumed by the sweep (R9: lagged)
//   thetaP/QP [class][n_pos]     deviational temperature / heat source permuted into each class's sweep order
//   part   [class][5][n_pos]     per-class partial moments (A1, A2, qx, qy, qz)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/nanobte.h"

#define NB_MAX_CLASSES 8  // structured: octants (quadrants in 2-D)

// ---- per-octant tables of the structured sweep -------------------------------------------------------------
// Pencils (lines of cells along the sweep axis u) of a class are sorted by (m = v'+w', w'); the pencil index p is
// also the pencil's slot in the shared-memory wavefront state.  Each diagonal m is padded to an even number of slots
// (padding slots are holes), so hyperplane h = u'+v'+w' holds the contiguous slot range [lo, lo+cnt) with lo and cnt
// even and lives at positions start + (p - lo) of every e row of the class; start is a multiple of 16 cells.  Both
// the per-plane table segments and the state-row segment that is the plane's output are therefore legal 1-D bulk
// TMA transfers (16-byte aligned, multiple of 16 bytes).  The class's boundary-inflow row is ordered by consuming
// hyperplane, each plane's slice [in_lo(h), in_lo(h+1)) padded to an even length for the same reason.
struct OctTab {
  const uint2 *pen;          // [n_pen]   .x = m, .y = pencil index of the v-upwind pencil | w-upwind pencil << 16 (n_pen = none)
  const int4 *plane;         // [H+1][2]  {wall lo, wall cnt, interior lo, interior cnt}, {start, in_lo, q_lo, 0}; entry H is the
                             //           sentinel {0,0,0,0}, {n_pos, n_in, n_q, 0}
  const double2 *tq;         // [n_pos+16] per position in sweep order: .x = theta, .y = bit pattern of a 64-bit record:
                             //   bit 0..2 u/v/w upwind value is a boundary inflow, bit 3 hole / padding, bit 4 source cell,
                             //   bits 5..17 first inflow index - in_lo(h), bits 18..31 index into the plane's qlist slice,
                             //   bits 32..47 slot of the v-upwind pencil, bits 48..63 slot of the w-upwind pencil
  const double *qlist;       // Qdot of the source cells in sweep order; hyperplane h owns [q_lo(h), q_lo(h+1)), even length
  const double *rhu;         // [nu]      1/h_u in primed coordinates (non-uniform spacing only)
  const double2 *pen_rh;     // [n_pen]   (1/h_v, 1/h_w) of the pencil (non-uniform spacing only)
  int64_t bin_base;          // offset of the class's first inflow row in bin
  int32_t n_pen, H, n_pos, n_in, row0, n_rows, p_max;
};

struct SweepArgs {
  const int32_t *task_oct;   // [n_tasks]
  const int32_t *task_row;   // [n_tasks] first row of the task, relative to the class's row0
  const double *coef;        // [rows][8]  uniform: k_theta,k_Q,c_u,c_v,c_w ; general: A,S,1/tau,v|s_u|,v|s_v|,v|s_w|
  const double *bin;         // inflow rows: class c, local row k at bin_base[c] + k * n_in[c]
  double *e;                 // [rows][e_stride]
  int64_t e_stride;
  int32_t nu, sp, pcap, gcap, qcap;  // pencil length, state pitch (>= n_pen + 1, even), table stage capacity in cells
                             // (multiple of 4), inflow / source stage capacities in values (even)
};

// ---- boundary-closure kernel ----------------------------------------------------------------------------------
struct BoundaryArgs {
  int32_t n_bf, B, D, n_cls;
  const int32_t *bf_act;      // [n_bf] owner (active index)
  const int32_t *bf_type;     // [n_bf]
  const double *bf_p, *bf_den, *bf_area, *bf_eps_w;  // bf_eps_w = (T_w - T_ref)/W for thermalizing faces
  const double *bf_sn;        // [n_bf][D]  s_d . n_f
  const int32_t *bf_mirror;   // [n_bf][D]  mirrored direction for incoming d (specular/mixed) or -1
  const int32_t *bf_inidx;    // [n_bf][D]  index of this face in direction d's inflow row, -1 if not incoming
  const int32_t *bf_opos;     // [n_bf][D]  position of the owner cell in direction d's e row (outgoing d), else -1
  const int32_t *dir_row0;    // [D]        e row of (direction d, band 0); band b is row dir_row0[d] + b
  const double *w, *C, *v;
  const int64_t *dir_bin;     // [D] base offset of direction d in bin
  const int32_t *dir_nin;     // [D] inflow row length of direction d
  const double *e;
  int64_t e_stride;
  double *bin, *G, *faceflux; // G [n_bf][B], faceflux [n_bf][B] = v_b sum_i w_i (s_i.n) eps_face
};

struct nanobte_solver {
  int kind = 0;  // 0 structured, 1 unstructured
  int dim = 0, n_cells = 0, n_act = 0, B = 0, D = 0, n_bf = 0, n_tags = 0, n_cls = 0;
  double T_ref = 0, W = 0, beta = 0, Csum = 0, kappa = 0, cg_rtol = 1e-12;
  int cg_max_iter = 100000;
  bool any_therm = false;
  cudaStream_t stream = nullptr;
  // second stream of the library's own (tile-dataflow path): the moment combine + update runs beside the closure kernels of the
  // same iteration (they touch disjoint data); forked and joined with the two events inside nanobte_update_temperature
  cudaStream_t aux_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  int n_sm = 148;

  // device arena
  char *arena = nullptr;
  size_t arena_bytes = 0;
  bool arena_owned = false;

  // host copies needed at run time
  std::vector<int32_t> h_bf_tag;
  std::vector<double> h_C;

  // structured sweep
  SweepArgs sw{};
  int sweep_G = 1, sweep_threads = 0, sweep_rmax = 1, n_tasks = 0, pencil_axis = 0, n_planes = 0, sweep_variant = 3, sweep_rp = 0;
  bool uniform = true;
  const OctTab *d_octs = nullptr;
  size_t sweep_smem = 0;
  int64_t n_pos = 0, n_inflow = 0, e_stride = 0;

  // tile-dataflow sweep with fused moments (brick.h); non-null = this path is the solver's sweep
  struct BrickState *brick = nullptr;
  // multigrid-preconditioned CG (cg_mg.h); non-null = the synthetic correction uses it
  struct MgPlan *mg = nullptr;
  bool keep_e = true;  // nanobte_sweep stores the distribution (nanobte_set_keep_e)

  // unstructured sweep (see sweep_unstructured.cu)
  struct UnsArgs *uns = nullptr;
  bool uns_staged = false;

  BoundaryArgs bd{};
  // structured grids: closures split into a G/flux kernel over reflecting faces and an inflow-cache kernel
  bool split_closures = false, therm_stale = true, swept_since_closure = false;
  const int32_t *cls_inbf[NB_MAX_CLASSES] = {nullptr};  // per class: face id per inflow slot (-1 = padding)
  int32_t cls_nin[NB_MAX_CLASSES] = {0}, cls_ndirs[NB_MAX_CLASSES] = {0};
  const int32_t *cls_dirs = nullptr;                     // [n_cls][max_cls_dirs]
  int max_cls_dirs = 0;
  const int32_t *cls_outbf[NB_MAX_CLASSES] = {nullptr}, *cls_outpos[NB_MAX_CLASSES] = {nullptr};  // outgoing wall cells per class
  const uint8_t *cls_outord[NB_MAX_CLASSES] = {nullptr}, *bf_nord = nullptr;
  int32_t cls_nout[NB_MAX_CLASSES] = {0};
  double *g_partial = nullptr;                            // [4][n_bf][B] per-class shares of gnum
  const int32_t *refl_faces = nullptr, *therm_faces = nullptr;
  int n_refl = 0, n_therm = 0;

  // moments / update
  int32_t *cls_npos_h = nullptr;
  int32_t cls_npos[NB_MAX_CLASSES] = {0};
  int32_t cls_nsys[NB_MAX_CLASSES] = {0};  // e rows of class c: [cls_row0[c], cls_row0[c] + cls_nsys[c])
  int32_t cls_row0[NB_MAX_CLASSES] = {0};
  const double *mcoef = nullptr;         // [rows][5]  w/tau, w, v w sx, v w sy, v w sz
  double *part = nullptr;                // [n_cls][5][e_stride]
  const int32_t *a2pos = nullptr;        // [n_cls][n_act]
  const int32_t *dir_cls = nullptr;      // [D] class of each direction
  double2 *tq[NB_MAX_CLASSES] = {nullptr};
  double *theta = nullptr, *theta_prev = nullptr, *theta_SI = nullptr, *theta_en = nullptr, *q = nullptr;  // [n_act]
  const double *Qdot = nullptr;          // [n_act]
  const int32_t *act2cell = nullptr, *cell2act = nullptr;
  unsigned long long *d_maxdT = nullptr; // bit pattern of a non-negative double
  double *h_pinned = nullptr;            // pinned host scratch (8 doubles)

  // diffusion / CG
  const int32_t *cg_nbr = nullptr;       // [6 or maxf][n_act]
  const double *cg_coef = nullptr;       // [nf][n_act]
  const double *cg_diag = nullptr, *vol = nullptr;
  const int32_t *cellbf_ptr = nullptr, *cellbf = nullptr;  // CSR: reflecting boundary faces of each active cell
  const double *fourier_rhs = nullptr;   // [n_act] right-hand side of the Fourier initial guess (R21)
  const double *cg_rhs_direct = nullptr; // non-null: the CG kernels take this right-hand side instead of R14c/R14c'
  double *leak_sum = nullptr;            // [n_bf] band shards: the R14c' leak summed over ALL bands (nanobte_import_moments)
  bool leak_imported = false;            // the CG takes leak_sum instead of summing its own bands' face fluxes
  int cg_nf = 0;
  double *cg_x = nullptr, *cg_r = nullptr, *cg_p0 = nullptr, *cg_p1 = nullptr, *cg_rhs = nullptr, *cg_scal = nullptr;
  double *cg_partial = nullptr;
  int cg_blocks = 0;
  // fused CG (cg.cu, cg_fused_kernel): cells cut into one contiguous chunk per CTA, vectors on chip
  bool cgf_ok = false, cg_force_generic = false, cgf_uni = false;
  double cgf_cfu[6] = {0, 0, 0, 0, 0, 0};
  bool cgf_recycle = true;              // Galerkin initial guess from the last two CG solutions
  int cgf_nprev = 0;
  double *cgf_xprev = nullptr, *cgf_gpart = nullptr;  // face-uniform stencil coefficients (cgf_uni)
  int cgf_nblk = 0, cgf_chunk = 0, cgf_cpt = 0, cgf_nh_cap = 0;
  size_t cgf_smem = 0;
  const int32_t *cgf_perm = nullptr;   // [n] CG index -> active cell index (spatially compact chunks)
  const double *cgf_coef = nullptr, *cgf_diag = nullptr;  // stencil in CG order
  const int32_t *cgf_nloc = nullptr;   // [nf][n] index of the neighbour inside its owner CTA's local vector
  const int32_t *cgf_hptr = nullptr;   // [nblk+1] halo lists
  const int32_t *cgf_hidx = nullptr;   // global cell index of every halo entry
  double *cgf_w = nullptr;             // [2][n]   A r, published every iteration (double buffered)
  double *cgf_part = nullptr;          // [2][nblk][2] per-CTA partial dot products (double buffered)
  unsigned int *cgf_bar = nullptr;     // grid barrier counter

  // boundary heat
  const int32_t *tagface_ptr = nullptr, *tagface = nullptr;  // CSR faces per tag
  double *d_tagheat = nullptr;

  std::vector<double> hist_dT;
  std::vector<int32_t> hist_cg;
  int64_t launches = 0;
  std::string err;
};

// error helpers ------------------------------------------------------------------------------------------------
int nb_fail(nanobte_solver *h, int code, const char *fmt, ...);
#define NB_CUDA(h, call)                                                                              \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess) return nb_fail((h), NANOBTE_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

// kernels_common.cu
int nb_launch_boundary(nanobte_solver *h, int init = 0);
int nb_launch_gcomb(nanobte_solver *h, const int32_t *faces, int n_faces, const uint8_t *nord);
int nb_refresh_thermalizing(nanobte_solver *h);
int nb_launch_moments(nanobte_solver *h);
int nb_launch_update(nanobte_solver *h, int mode /*0: theta<-theta_SI, 1: theta<-theta_SI+x*/);
int nb_launch_get_e(nanobte_solver *h, int b0, int nb, int d0, int nd, double *dst_dev, int deviational);
int nb_launch_scatter_cells(nanobte_solver *h, const double *src_act, double *dst_cells, int ncomp, double add);
int nb_launch_set_theta(nanobte_solver *h, const double *T_cells_dev);
int nb_launch_tagheat(nanobte_solver *h);
int nb_launch_leak_sum(nanobte_solver *h);
int nb_cg_solve(nanobte_solver *h, int *iters);
int nb_cg_blocks(nanobte_solver *h);
// sweep_structured.cu
int nb_launch_sweep_structured(nanobte_solver *h);
int nb_sweep_structured_config(nanobte_solver *h, int n_pen_max, int p_max, int gcap, int qcap, int H, int want_G, int want_threads,
                               int n_sys_min_class, int want_variant, int n_sys_total);
// sweep_unstructured.cu
int nb_launch_sweep_unstructured(nanobte_solver *h);
void nb_free_unstructured(nanobte_solver *h);
