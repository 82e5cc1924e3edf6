// brick.h -- private declarations of the tile-dataflow sweep with fused moments (DESIGN.md
// "Brick sweep").  3-D structured grids with uniform spacing.
//
// Decomposition.  The grid cross-section (the two axes other than the pencil axis u) is cut into tiles of at most
// 8 x 8 pencils (cuts follow the mask, so that walls fall on tile edges), the pencil axis into segments.  A task is
// (octant class c, band group g, tile, segment): one CTA, ONE THREAD PER (band, direction) SYSTEM of the group, walks
// the task's cells in the upwind-lexicographic order (u', w', v'), every thread doing the forward substitution of its own
// system.  There is no wavefront inside a task and no barrier in the substitution: the u-upwind value comes from a
// per-system plane buffer in shared memory ([cell of the tile][system], the previous u-plane), the v- and w-upwind values
// stay in registers.  After every u-plane the CTA switches roles once: lanes become cells and reduce the plane buffer over
// the systems to the five moment partials (Eq. 5, R13, Eq. 7) -- the distribution never goes to HBM unless asked for.
// Tasks exchange tile-face values through global memory (L2) in a dataflow: a task publishes a progress counter per
// u-plane (release), its two downstream tiles acquire it one plane behind.  Tasks are handed out in topological
// order by a ticket counter, so a waiting CTA only ever waits for a CTA that is already running.
//
// Row spaces (every row holds the S_g systems of group g of class c at a pitch of kBrickRow doubles, lanes = systems:
// every access is coalesced):
//   inflow rows of class c   per task: FU [64] (u-face of the segment), FV [nu][8], FW [nu][8] (v- / w-face, one row per
//                            cell of the face and u-plane), IRR [n_irr] (walls inside the tile, consumption order).
//                            Written by the upstream task (interior tile faces) or by the closure kernel (boundary
//                            faces, lagged: R9) -- exactly one producer per row.
//   wall rows of class c     eps of every cell with an outgoing boundary face, task by task in sweep order (closures).
//   cell positions           pos = pos0(task) + 64 * u_local + 8 * w_local + v_local  (theta/Qdot/flags per class;
//                            moment partials and, on request, eps per (class, group)).
#pragma once
#include "internal.h"

constexpr int kBrickTile = 8;          // tile edge (pencils)
constexpr int kBrickCells = 64;        // cells per u-plane of a tile
constexpr int kBrickMaxS = 128;        // systems per task = threads per CTA
constexpr int kBrickRow = 128;         // pitch in doubles of every inflow / wall / eps row (compile-time: row addresses are immediates)
constexpr int kBrickPitch = 129;       // plane-buffer row pitch in doubles (odd: lanes = cells is conflict-free too)

enum : uint8_t {
  BRK_ACT = 1,      // active cell
  BRK_INJ_U = 2,    // u-upwind neighbour is a wall INSIDE the segment: next row of the IRR stream
  BRK_INJ_V = 4,    // same for v (v_local > 0)
  BRK_INJ_W = 8,    // same for w (w_local > 0)
  BRK_SRC = 16,     // Qdot != 0
  BRK_WALL = 32     // has an outgoing boundary face for this class: eps goes to the next wall row
};

// How a task learns that the rows of an inflow face are there.
//   BOUNDARY  no upstream task: closure rows, written before the launch.
//   TAGGED    every row of the face is written by the upstream task.  The least significant mantissa bit of a value that
//             crosses a tile face carries the parity of the sweep (a relative perturbation of at most 2.2e-16, below the
//             rounding of the substitution itself), so the value is its own ready flag: no fence, no counter, no poll
//             separate from the load; a stale row (last sweep's) has the other parity and is simply loaded again.
//   COUNTER   the face mixes rows of the upstream task with closure rows (walls inside a tile face): the upstream task
//             publishes a progress counter with release semantics after every plane (BrickTask::publish), this task
//             acquires it.
enum : int32_t { BRK_FACE_BOUNDARY = 0, BRK_FACE_TAGGED = 1, BRK_FACE_COUNTER = 2 };

struct BrickTask {
  int32_t cg;                  // (class, group) index
  int32_t nu, tv, tw;          // planes, tile width (v), tile height (w)
  int32_t pos0;                // first cell position
  int32_t fu0, fv0, fw0, ir0;  // inflow rows of this task
  int32_t wo0;                 // first wall row of this task
  int32_t up_u, up_v, up_w;    // tasks whose outflow this task consumes (-1: none -- the rows are boundary values)
  int32_t dn_fu0, dn_fv0, dn_fw0;  // inflow rows of the downstream tasks this task feeds (-1: none)
  int32_t plain;               // 1: every cell of the tv x tw x nu box is active (no wall inside the box): straight-line path
  uint32_t src_lo, src_hi;     // bit u: plane u of the task holds a cell with Qdot != 0 (nu <= 64)
  int32_t wall_any;            // the task has cells with an outgoing boundary face
  int32_t fv_mode, fw_mode;    // how the v- / w-face inflow rows become valid: BRK_FACE_*
  int32_t publish;             // a downstream task follows this one through the progress counter: publish every plane
  int32_t wu0, wv0, ww0;       // wall rows as face blocks (first row or -1): what the u- / v- / w-face stores go to where there
                               // is no downstream tile but a wall (tasks whose faces are each all wall or all interior)
  int32_t pad[2];
};
static_assert(sizeof(BrickTask) == 112, "BrickTask layout");

struct BrickCG {
  int32_t cls, S, nb, nd;      // class, systems (= nb * nd), bands, directions of the class; system = band_local * nd + dir_local
  int32_t b0, pad;
  int64_t inf_base, wall_base, part_base, e_base;  // offsets in doubles of this (class, group)'s blocks
  int64_t coef_base;           // [S][5] sweep coefficients, then [nd][4] (w, w s), then [nb][2] (1/tau, v)
};

constexpr int kBrickInRows = 4;  // records per batch of the fast inflow kernel (one face type per batch)

// One boundary-inflow row of a class, everything the closure kernel needs about it in one 16-byte load.
struct BrickInRow {
  int32_t bf;          // boundary face
  int32_t row;         // inflow row (of every group of the class)
  int32_t msrc;        // wall row, in the mirror class, of the cell the specular part comes from (-1: none)
  uint8_t type, cm, perm, pad;  // face type; mirror class; which direction permutation of the class (BrickState::in_perm)
};

// One outgoing-face entry of a class (gsum kernel): the face, its wall row (of every group of the class), the class's rank
// among the face's outgoing classes and the face type in one 16-byte load.
struct BrickOutRow {
  int32_t bf, row;
  uint8_t ord, type, pad[6];
};

struct BrickArgs {
  const BrickTask *tasks;      // in launch (topological) order
  const BrickCG *cgs;
  int32_t n_tasks, store_e;
  uint32_t parity;             // of this sweep (alternates; the rows start as zeros, so the first sweep has parity 1)
  const double *th[NB_MAX_CLASSES];     // per class [npos] theta (sweep order; refreshed by the update kernel)
  const double *qd[NB_MAX_CLASSES];     // per class [npos] Qdot
  const uint8_t *flg[NB_MAX_CLASSES];   // per class [npos]
  int32_t npos[NB_MAX_CLASSES];         // positions per class (partials are [5][npos] per (class, group))
  int32_t scratch_row[NB_MAX_CLASSES];  // per class: first of 8 inflow rows that no task reads (v-face rows of boundary tiles)
  double *inf, *wall, *part, *e;
  const double *coef;
  unsigned int *ticket;        // [1] next task
  unsigned int *prog;          // [n_tasks] u-planes completed (published with release semantics)
};

// Everything the brick path keeps in the solver.
struct BrickState {
  BrickArgs a{};
  int n_cg = 0, n_groups = 0, grid = 0;
  size_t smem = 0;
  int64_t inf_total = 0, wall_total = 0, part_total = 0, e_total = 0;
  bool e_valid = false;        // the last sweep stored eps
  uint32_t parity = 0;         // of the last sweep
  // closures
  const int32_t *in_row[NB_MAX_CLASSES] = {nullptr}, *in_bf[NB_MAX_CLASSES] = {nullptr};  // boundary-inflow rows of a class
  int32_t n_in[NB_MAX_CLASSES] = {0};
  const int32_t *out_bf[NB_MAX_CLASSES] = {nullptr}, *out_row[NB_MAX_CLASSES] = {nullptr};  // outgoing faces of a class, wall row of their cell
  const uint8_t *out_ord[NB_MAX_CLASSES] = {nullptr}, *bf_nord = nullptr;
  int32_t n_out[NB_MAX_CLASSES] = {0};
  int s_max = 0;
  const int32_t *bf_wrow = nullptr;                    // [n_cls][n_bf] wall row of the face's cell in class c, -1 if not outgoing
  const int32_t *dir_local = nullptr;                  // [D] index of a direction inside its class
  const int32_t *cg_of = nullptr;                      // [n_cls][B] (class, band) -> cg
  const int32_t *a2pos = nullptr;                      // [n_cls][n_act]
  const int32_t *pos2a = nullptr;                      // [npos of class 0]
  const BrickOutRow *out_rec[NB_MAX_CLASSES] = {nullptr};  // per class [n_out]: records of the gsum kernel
  const BrickInRow *in_rec[NB_MAX_CLASSES] = {nullptr};  // per class [n_rec]: records of the fast inflow kernel, by type
  int32_t n_rec[NB_MAX_CLASSES] = {0};
  const uint8_t *in_perm = nullptr;                    // [n_cls][8][16] direction -> mirrored direction (local indices; 255: none)
  int32_t cg0[NB_MAX_CLASSES] = {0};                   // first (class, group) of a class
  bool in_fast = false;                                // the records are valid (same band groups in every class, <= 8 permutations)
  double *th[NB_MAX_CLASSES] = {nullptr};
};

// sweep_brick.cu
int nb_launch_sweep_brick(nanobte_solver *h, int store_e);
size_t nb_brick_smem_bytes();
// closures_brick.cu
int nb_brick_closures(nanobte_solver *h, int init);
int nb_brick_refresh_thermalizing(nanobte_solver *h);
int nb_brick_update(nanobte_solver *h, int mode);
int nb_brick_set_theta(nanobte_solver *h, const double *T_cells_dev);
int nb_brick_get_e(nanobte_solver *h, int b0, int nb, int d0, int nd, double *dst_dev, int deviational);
void nb_free_brick(nanobte_solver *h);
