// brick_host.h -- host-side tables of the tile-dataflow sweep (setup_brick.cu), private to csrc/.
#pragma once
#include <vector>

#include "brick.h"
#include "host_util.h"

// What setup_structured.cu has already worked out about the problem.
struct BrickCtx {
  int n[3];                         // grid
  const uint8_t *act;               // [n_cells]
  int pa, va, wa;                   // pencil axis and the two cross-section axes
  int ncls;
  int sign[NB_MAX_CLASSES][3];      // sweep direction of every class along x, y, z
  std::vector<std::vector<int>> dirs;  // directions of every class, class order
  const int32_t *facebf;            // [n_cells][6] boundary face of (cell, side) or -1
  const Common *cm;
  const GenericTables *G;
  const double *coef;               // [rows][8] uniform-spacing sweep coefficients, row = cls_row0[c] + dir_local * B + b
  const int32_t *cls_row0;
  const double *Qdot, *T_init;      // [n_cells] or NULL
  double T_ref;
};

struct BrickHost {
  struct Cls {
    std::vector<double> th, qd;
    std::vector<uint8_t> flg;
    std::vector<int32_t> in_row, in_bf;             // boundary-inflow rows and their faces
    std::vector<int32_t> out_bf, out_row;           // outgoing faces and the wall row of their cell, wall-row order
    std::vector<uint8_t> out_ord;                   // rank of the class among the face's outgoing classes
    std::vector<BrickOutRow> out_rec;               // records of the gsum kernel
    std::vector<BrickInRow> in_rec;                 // records of the fast inflow kernel
    int npos = 0, nrow = 0, nwall = 0, scratch_row = 0;
  };
  int ncls = 0;
  std::vector<Cls> cls;
  std::vector<BrickTask> tasks;
  std::vector<BrickCG> cgs;
  std::vector<double> coef;
  std::vector<int32_t> cg_of, dir_local, bf_wrow, a2pos;
  std::vector<uint8_t> bf_nord, in_perm;
  std::vector<int32_t> cg0;
  bool in_fast = false;
  int64_t inf_total = 0, wall_total = 0, part_total = 0, e_total = 0;
};

int nb_brick_build(nanobte_solver *h, const BrickCtx &x, BrickHost &bh);
int nb_brick_upload(nanobte_solver *h, Arena &A, BrickHost &bh);
