// host_util.h -- host-side helpers of libnanobte: device arena with a dry (size-counting) pass, validation
// shared by the structured and unstructured create paths.  Private to csrc/.
#pragma once
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "internal.h"

// Bump allocator over one device block.  Pass 1 (dry) only counts; pass 2 copies.
struct Arena {
  nanobte_solver *h;
  bool dry;
  size_t off = 0;
  int rc = 0;
  Arena(nanobte_solver *h_, bool dry_) : h(h_), dry(dry_) {}
  void *raw(size_t bytes) {
    size_t a = (off + 255) & ~size_t(255);
    off = a + bytes;
    if (dry) return nullptr;
    if (off > h->arena_bytes) {
      rc = NANOBTE_E_ALLOC;
      return nullptr;
    }
    return h->arena + a;
  }
  template <class T>
  T *put(const std::vector<T> &v) {
    T *p = (T *)raw(v.size() * sizeof(T) + 16);
    if (!dry && p && !v.empty()) {
      cudaError_t e = cudaMemcpyAsync(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, h->stream);
      if (e != cudaSuccess) rc = NANOBTE_E_CUDA;
    }
    return p;
  }
  template <class T>
  T *zeros(size_t n) {
    T *p = (T *)raw(n * sizeof(T) + 16);
    if (!dry && p) {
      cudaError_t e = cudaMemsetAsync(p, 0, n * sizeof(T) + 16, h->stream);
      if (e != cudaSuccess) rc = NANOBTE_E_CUDA;
    }
    return p;
  }
};

// Validated copies of the band table / quadrature / tags and the scalars derived from them.
struct Common {
  int B = 0, D = 0, dim = 0, n_tags = 0;
  std::vector<double> C, v, tau, share, s, w;
  std::vector<int> tag_type;
  std::vector<double> tag_T;
  double W = 0, beta = 0, Csum = 0, kappa = 0;
};

int nb_validate_common(nanobte_solver *h, int dim, const nanobte_bands *bands, const nanobte_quadrature *quad,
                       const nanobte_tag *tags, int n_tags, Common &c);
int nb_check_device(nanobte_solver *h);
void nb_query_sm_count(nanobte_solver *h);
// Finds j with s_j == s_d - 2 (s_d.n) n  (squared distance < 1e-18), or -1.
int nb_find_mirror(const Common &c, int d, const double n[3]);

// Everything both mesh kinds upload after their own geometry pass (boundary tables, moments, CG, tags).
struct GenericTables {
  // per boundary face
  std::vector<int32_t> bf_act, bf_type;
  std::vector<double> bf_p, bf_den, bf_area, bf_eps_w, bf_sn;
  std::vector<int32_t> bf_mirror, bf_inidx, bf_opos;
  // per direction
  std::vector<int64_t> dir_bin;
  std::vector<int32_t> dir_nin, dir_row0;
  // moments
  std::vector<double> mcoef;
  // cells
  std::vector<int32_t> act2cell, cell2act;
  std::vector<double> vol, Qdot_act, theta0;
  // CG (ELL, nf faces per cell)
  int cg_nf = 0;
  std::vector<int32_t> cg_nbr;
  std::vector<double> cg_coef, cg_diag;
  std::vector<int32_t> cellbf_ptr, cellbf;
  std::vector<double> fourier_rhs;  // [n] right-hand side of the Fourier initial guess (R21): V Qdot + sum_thermalizing kappa A_f (T_w - T_ref) / d_cf
  std::vector<double> cg_xyz;      // [n][3] cell centres in any consistent unit (partitioning of the CG only)
  int cg_grid[3] = {0, 0, 0};      // structured grids: lattice dimensions, cg_xyz holds the integer lattice coordinates
  std::vector<int32_t> tagface_ptr, tagface;
  int64_t bin_total = 0;
};
int nb_upload_generic(nanobte_solver *h, Arena &A, const Common &c, GenericTables &g);
