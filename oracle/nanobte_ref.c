/*
 * nanobte_ref.c -- CPU fp64 ORACLE (test infrastructure; see nanobte_ref.h for scope, citations
 * and the list of pins).  Plain loops over a generic face-based finite-volume mesh; the only
 * parallelism is an OpenMP "parallel for" over the independent direction tasks.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC nanobte_ref.c -o libnanobte_ref.so -lm
 */
#include "nanobte_ref.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct nanobte_ref {
  int dim, n_cells, n_act;
  int *act2cell, *cell2act;
  /* faces of active cell a: fptr[a] .. fptr[a+1]-1 */
  int *fptr, *fnbr, *fbf;
  double *farea, *fnrm, *fdist, *vol;
  int nf;
  /* bands, quadrature */
  int B, D;
  double *C, *v, *tau, *share, *s, *w;
  double W, beta, Csum, kappa;
  /* boundary faces (user order) */
  int n_bf;
  int *bf_tag, *bf_act, *bf_face, *bf_mirror;
  double *bf_p, *bf_den;
  int n_tags;
  int *tag_type;
  double *tag_T;
  /* upwind-first cell order per direction: order[i*n_act + k] */
  int *order;
  /* state (deviational) */
  double T_ref;
  double *Qdot, *theta, *theta_prev, *theta_SI, *theta_en, *q;
  double *eps; /* [B][D][n_act] */
  double *G;   /* [n_bf][B]     */
  double *bcv; /* [n_bf][B][D]  */
  double cg_rtol;
  int cg_max_iter;
  double *hist_dT;
  int *hist_cg;
  int n_hist, cap_hist;
  int n_threads;
  char err[256];
};

#define FAIL(h, code, ...)                              \
  do {                                                  \
    snprintf((h)->err, sizeof((h)->err), __VA_ARGS__);  \
    return (code);                                      \
  } while (0)

static double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* ------------------------------------------------------------------------------------------ */
/* setup shared by both mesh kinds (everything that is iteration independent)     */
/* ------------------------------------------------------------------------------------------ */
static int finish_setup(nanobte_ref *h, int B, const double *C, const double *v, const double *tau,
                        const double *share, int D, const double *s, const double *w, int n_tags,
                        const int32_t *tag_type, const double *tag_T, const double *Qdot, double T_ref,
                        const double *T_init, double cg_rtol, int cg_max_iter) {
  int na = h->n_act;
  if (B < 1 || D < 1 || n_tags < 0) FAIL(h, NBR_E_INVALID, "B, D must be >= 1");
  h->B = B;
  h->D = D;
  h->C = malloc(sizeof(double) * B);
  h->v = malloc(sizeof(double) * B);
  h->tau = malloc(sizeof(double) * B);
  h->share = malloc(sizeof(double) * B);
  h->s = malloc(sizeof(double) * 3 * D);
  h->w = malloc(sizeof(double) * D);
  h->n_tags = n_tags;
  h->tag_type = malloc(sizeof(int) * (n_tags > 0 ? n_tags : 1));
  h->tag_T = malloc(sizeof(double) * (n_tags > 0 ? n_tags : 1));
  if (!h->C || !h->v || !h->tau || !h->share || !h->s || !h->w || !h->tag_type || !h->tag_T)
    FAIL(h, NBR_E_ALLOC, "alloc");
  h->Csum = 0.0;
  h->beta = 0.0;
  for (int b = 0; b < B; ++b) {
    if (!(C[b] > 0) || !(v[b] > 0) || !(tau[b] > 0)) FAIL(h, NBR_E_INVALID, "band %d: C, v, tau must be > 0", b);
    h->C[b] = C[b];
    h->v[b] = v[b];
    h->tau[b] = tau[b];
    h->Csum += C[b];
    h->beta += C[b] / tau[b]; /* denominator of Eq. 5 */
  }
  for (int b = 0; b < B; ++b) h->share[b] = share ? share[b] : C[b] / h->Csum;
  h->W = 0.0; /* W_Omega = sum_i w_i, Eq. 11 */
  double ws[3] = {0, 0, 0}, tr = 0.0;
  for (int i = 0; i < D; ++i) {
    if (!(w[i] > 0)) FAIL(h, NBR_E_QUADRATURE, "weight %d not positive", i);
    double nn = sqrt(dot3(s + 3 * i, s + 3 * i));
    if (fabs(nn - 1.0) > 1e-12) FAIL(h, NBR_E_QUADRATURE, "direction %d is not a unit vector", i);
    h->w[i] = w[i];
    for (int k = 0; k < 3; ++k) {
      h->s[3 * i + k] = s[3 * i + k];
      ws[k] += w[i] * s[3 * i + k];
    }
    h->W += w[i];
    for (int k = 0; k < h->dim; ++k) tr += w[i] * s[3 * i + k] * s[3 * i + k];
  }
  for (int k = 0; k < h->dim; ++k)
    if (fabs(ws[k]) > 1e-12 * h->W) FAIL(h, NBR_E_QUADRATURE, "sum_i w_i s_i != 0 (component %d: %g)", k, ws[k]);
  /* kappa_bulk (R14d): kinetic value with the isotropic part of the discrete second angular moment,
   *   kappa = sum_b C_b v_b^2 tau_b * trace_dim(sum_i w_i s_i s_i^T) / (dim W)
   * = (1/3) sum C v^2 tau for unit vectors in 3-D, (1/2) sum C v^2 tau for in-plane unit vectors in 2-D. */
  h->kappa = 0.0;
  for (int b = 0; b < B; ++b) h->kappa += C[b] * v[b] * v[b] * tau[b];
  h->kappa *= tr / (h->dim * h->W);
  for (int t = 0; t < n_tags; ++t) {
    if (tag_type[t] < 0 || tag_type[t] > 3) FAIL(h, NBR_E_INVALID, "tag %d: unknown type %d", t, tag_type[t]);
    h->tag_type[t] = tag_type[t];
    h->tag_T[t] = tag_T[t];
  }
  /* every face without a neighbour must carry a boundary tag */
  for (int a = 0; a < na; ++a)
    for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f)
      if (h->fnbr[f] < 0 && h->fbf[f] < 0)
        FAIL(h, NBR_E_UNTAGGED, "cell %d has an exposed face without a boundary tag", h->act2cell[a]);
  /* per boundary face: incoming half-range sum (R7) and specular mirror map (O3) */
  h->bf_den = calloc(h->n_bf > 0 ? h->n_bf : 1, sizeof(double));
  h->bf_mirror = malloc(sizeof(int) * (size_t)(h->n_bf > 0 ? h->n_bf : 1) * D);
  if (!h->bf_den || !h->bf_mirror) FAIL(h, NBR_E_ALLOC, "alloc");
  for (int bf = 0; bf < h->n_bf; ++bf) {
    if (h->bf_tag[bf] < 0 || h->bf_tag[bf] >= n_tags) FAIL(h, NBR_E_INVALID, "boundary face %d: bad tag", bf);
    const double *n = h->fnrm + 3 * h->bf_face[bf];
    int type = h->tag_type[h->bf_tag[bf]];
    double den = 0.0;
    for (int i = 0; i < D; ++i) {
      double sn = dot3(h->s + 3 * i, n);
      h->bf_mirror[(size_t)bf * D + i] = -1;
      if (sn < 0) den += h->w[i] * (-sn);
      if (sn < 0 && (type == 2 || type == 3)) {
        double r[3];
        for (int k = 0; k < 3; ++k) r[k] = h->s[3 * i + k] - 2.0 * sn * n[k]; /* s - 2 (s.n) n */
        int found = -1;
        for (int j = 0; j < D && found < 0; ++j) {
          double d0 = h->s[3 * j] - r[0], d1 = h->s[3 * j + 1] - r[1], d2 = h->s[3 * j + 2] - r[2];
          if (d0 * d0 + d1 * d1 + d2 * d2 < 1e-18) found = j;
        }
        if (found < 0) FAIL(h, NBR_E_SPECULAR, "boundary face %d: mirror image of direction %d is not in the quadrature", bf, i);
        h->bf_mirror[(size_t)bf * D + i] = found;
      }
    }
    h->bf_den[bf] = den;
    if (h->bf_p[bf] < 0 || h->bf_p[bf] > 1) FAIL(h, NBR_E_INVALID, "boundary face %d: specularity outside [0,1]", bf);
  }
  /* upwind-first order per direction (Kahn); a leftover cell means a cyclic upwind graph (R16) */
  h->order = malloc(sizeof(int) * (size_t)D * na);
  int *indeg = malloc(sizeof(int) * na);
  if (!h->order || !indeg) FAIL(h, NBR_E_ALLOC, "alloc");
  for (int i = 0; i < D; ++i) {
    int *ord = h->order + (size_t)i * na;
    const double *si = h->s + 3 * i;
    for (int a = 0; a < na; ++a) {
      indeg[a] = 0;
      for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f)
        if (h->fnbr[f] >= 0 && dot3(si, h->fnrm + 3 * f) < 0) indeg[a]++;
    }
    int head = 0, tail = 0;
    for (int a = 0; a < na; ++a)
      if (indeg[a] == 0) ord[tail++] = a;
    while (head < tail) {
      int a = ord[head++];
      for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f) {
        int nb = h->fnbr[f];
        if (nb >= 0 && dot3(si, h->fnrm + 3 * f) > 0) { /* a is upwind of nb */
          if (--indeg[nb] == 0) ord[tail++] = nb;
        }
      }
    }
    if (tail != na) {
      free(indeg);
      FAIL(h, NBR_E_CYCLE, "upwind graph of direction %d is cyclic (%d of %d cells ordered)", i, tail, na);
    }
  }
  free(indeg);
  /* state */
  h->T_ref = T_ref;
  h->cg_rtol = cg_rtol > 0 ? cg_rtol : 1e-12;
  h->cg_max_iter = cg_max_iter > 0 ? cg_max_iter : 100000;
  h->Qdot = calloc(na, sizeof(double));
  h->theta = calloc(na, sizeof(double));
  h->theta_prev = calloc(na, sizeof(double));
  h->theta_SI = calloc(na, sizeof(double));
  h->theta_en = calloc(na, sizeof(double));
  h->q = calloc((size_t)na * 3, sizeof(double));
  h->eps = calloc((size_t)B * D * na, sizeof(double));
  h->G = calloc((size_t)(h->n_bf > 0 ? h->n_bf : 1) * B, sizeof(double));
  h->bcv = calloc((size_t)(h->n_bf > 0 ? h->n_bf : 1) * B * D, sizeof(double));
  if (!h->Qdot || !h->theta || !h->theta_prev || !h->theta_SI || !h->theta_en || !h->q || !h->eps || !h->G || !h->bcv)
    FAIL(h, NBR_E_ALLOC, "alloc of state failed");
  for (int a = 0; a < na; ++a) {
    h->Qdot[a] = Qdot ? Qdot[h->act2cell[a]] : 0.0;
    h->theta[a] = T_init ? T_init[h->act2cell[a]] - T_ref : 0.0; /* R12 */
  }
  h->cap_hist = 0;
  h->n_hist = 0;
  h->hist_dT = NULL;
  h->hist_cg = NULL;
#ifdef _OPENMP
  h->n_threads = omp_get_max_threads();
#else
  h->n_threads = 1;
#endif
  return NBR_OK;
}

static int copy_bf_meta(nanobte_ref *h, int n_bf, const int32_t *bf_tag, const double *bf_p) {
  h->n_bf = n_bf;
  size_t n = n_bf > 0 ? n_bf : 1;
  h->bf_tag = malloc(sizeof(int) * n);
  h->bf_p = calloc(n, sizeof(double));
  h->bf_act = malloc(sizeof(int) * n);
  h->bf_face = malloc(sizeof(int) * n);
  if (!h->bf_tag || !h->bf_p || !h->bf_act || !h->bf_face) return NBR_E_ALLOC;
  for (int i = 0; i < n_bf; ++i) {
    h->bf_tag[i] = bf_tag[i];
    h->bf_p[i] = bf_p ? bf_p[i] : 0.0;
    h->bf_act[i] = -1;
    h->bf_face[i] = -1;
  }
  return NBR_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* structured (optionally masked) grid -> generic faces                                         */
/* ------------------------------------------------------------------------------------------ */
int nanobte_ref_create_structured(int nx, int ny, int nz, const double *hx, const double *hy, const double *hz,
                                  const uint8_t *active, int n_bf, const int32_t *bf_cell, const uint8_t *bf_side,
                                  const int32_t *bf_tag, const double *bf_p, int B, const double *C,
                                  const double *v, const double *tau, const double *share, int D, const double *s,
                                  const double *w, int n_tags, const int32_t *tag_type, const double *tag_T,
                                  const double *Qdot, double T_ref, const double *T_init, double cg_rtol,
                                  int cg_max_iter, nanobte_ref **out) {
  if (!out) return NBR_E_INVALID;
  nanobte_ref *h = calloc(1, sizeof(*h));
  if (!h) return NBR_E_ALLOC;
  *out = h;
  if (nx < 1 || ny < 1 || nz < 1 || !hx || !hy || !hz) FAIL(h, NBR_E_INVALID, "bad grid");
  h->dim = nz > 1 ? 3 : 2;
  int nc = nx * ny * nz;
  h->n_cells = nc;
  h->cell2act = malloc(sizeof(int) * nc);
  if (!h->cell2act) FAIL(h, NBR_E_ALLOC, "alloc");
  int na = 0;
  for (int c = 0; c < nc; ++c) h->cell2act[c] = (!active || active[c]) ? na++ : -1;
  h->n_act = na;
  if (na == 0) FAIL(h, NBR_E_INVALID, "no active cell");
  h->act2cell = malloc(sizeof(int) * na);
  for (int c = 0; c < nc; ++c)
    if (h->cell2act[c] >= 0) h->act2cell[h->cell2act[c]] = c;
  int nside = 2 * h->dim;
  h->nf = na * nside;
  h->fptr = malloc(sizeof(int) * (na + 1));
  h->fnbr = malloc(sizeof(int) * h->nf);
  h->fbf = malloc(sizeof(int) * h->nf);
  h->farea = malloc(sizeof(double) * h->nf);
  h->fnrm = calloc((size_t)h->nf * 3, sizeof(double));
  h->fdist = malloc(sizeof(double) * h->nf);
  h->vol = malloc(sizeof(double) * na);
  if (!h->fptr || !h->fnbr || !h->fbf || !h->farea || !h->fnrm || !h->fdist || !h->vol) FAIL(h, NBR_E_ALLOC, "alloc");
  for (int a = 0; a < na; ++a) {
    int c = h->act2cell[a];
    int i = c % nx, j = (c / nx) % ny, k = c / (nx * ny);
    double dx = hx[i], dy = hy[j], dz = (h->dim == 3) ? hz[k] : 1.0; /* unit depth in 2-D */
    h->vol[a] = dx * dy * dz;
    h->fptr[a] = a * nside;
    for (int side = 0; side < nside; ++side) {
      int f = a * nside + side, axis = side / 2, sgn = (side & 1) ? 1 : -1;
      int ii = i + (axis == 0 ? sgn : 0), jj = j + (axis == 1 ? sgn : 0), kk = k + (axis == 2 ? sgn : 0);
      h->fnrm[3 * f + axis] = (double)sgn;
      h->farea[f] = (axis == 0) ? dy * dz : (axis == 1) ? dx * dz : dx * dy;
      double hc = (axis == 0) ? dx : (axis == 1) ? dy : dz;
      h->fbf[f] = -1;
      h->fnbr[f] = -1;
      h->fdist[f] = 0.5 * hc; /* centroid-to-face; replaced below for interior faces */
      if (ii >= 0 && ii < nx && jj >= 0 && jj < ny && kk >= 0 && kk < nz) {
        int cn = ii + nx * (jj + ny * kk);
        if (h->cell2act[cn] >= 0) {
          double hn = (axis == 0) ? hx[ii] : (axis == 1) ? hy[jj] : hz[kk];
          h->fnbr[f] = h->cell2act[cn];
          h->fdist[f] = 0.5 * (hc + hn); /* centroid-to-centroid */
        }
      }
    }
  }
  h->fptr[na] = na * nside;
  int rc = copy_bf_meta(h, n_bf, bf_tag, bf_p);
  if (rc) FAIL(h, rc, "alloc");
  for (int bf = 0; bf < n_bf; ++bf) {
    int c = bf_cell[bf], side = bf_side[bf];
    if (c < 0 || c >= nc || side >= nside || h->cell2act[c] < 0) FAIL(h, NBR_E_INVALID, "boundary face %d: bad cell/side", bf);
    int a = h->cell2act[c], f = a * nside + side;
    if (h->fnbr[f] >= 0) FAIL(h, NBR_E_INVALID, "boundary face %d is an interior face", bf);
    if (h->fbf[f] >= 0) FAIL(h, NBR_E_INVALID, "boundary face %d listed twice", bf);
    h->fbf[f] = bf;
    h->bf_act[bf] = a;
    h->bf_face[bf] = f;
  }
  return finish_setup(h, B, C, v, tau, share, D, s, w, n_tags, tag_type, tag_T, Qdot, T_ref, T_init, cg_rtol,
                      cg_max_iter);
}

/* ------------------------------------------------------------------------------------------ */
/* unstructured 2-D polygons (CCW) -> generic faces                                             */
/* ------------------------------------------------------------------------------------------ */
typedef struct {
  int lo, hi, face;
} edge_rec;
static int edge_cmp(const void *a, const void *b) {
  const edge_rec *x = a, *y = b;
  if (x->lo != y->lo) return x->lo < y->lo ? -1 : 1;
  if (x->hi != y->hi) return x->hi < y->hi ? -1 : 1;
  return x->face < y->face ? -1 : (x->face > y->face);
}

int nanobte_ref_create_unstructured(int n_nodes, const double *xy, int n_cells, const int32_t *cell_ptr,
                                    const int32_t *cell_nodes, int n_bf, const int32_t *bf_nodes,
                                    const int32_t *bf_tag, const double *bf_p, int B, const double *C,
                                    const double *v, const double *tau, const double *share, int D,
                                    const double *s, const double *w, int n_tags, const int32_t *tag_type,
                                    const double *tag_T, const double *Qdot, double T_ref, const double *T_init,
                                    double cg_rtol, int cg_max_iter, nanobte_ref **out) {
  if (!out) return NBR_E_INVALID;
  nanobte_ref *h = calloc(1, sizeof(*h));
  if (!h) return NBR_E_ALLOC;
  *out = h;
  if (n_nodes < 3 || n_cells < 1 || !xy || !cell_ptr || !cell_nodes) FAIL(h, NBR_E_INVALID, "bad mesh");
  h->dim = 2;
  h->n_cells = h->n_act = n_cells;
  int na = n_cells;
  h->cell2act = malloc(sizeof(int) * na);
  h->act2cell = malloc(sizeof(int) * na);
  for (int c = 0; c < na; ++c) h->cell2act[c] = h->act2cell[c] = c;
  h->nf = cell_ptr[na];
  h->fptr = malloc(sizeof(int) * (na + 1));
  h->fnbr = malloc(sizeof(int) * h->nf);
  h->fbf = malloc(sizeof(int) * h->nf);
  h->farea = malloc(sizeof(double) * h->nf);
  h->fnrm = calloc((size_t)h->nf * 3, sizeof(double));
  h->fdist = malloc(sizeof(double) * h->nf);
  h->vol = malloc(sizeof(double) * na);
  double *cen = malloc(sizeof(double) * 2 * na);
  edge_rec *er = malloc(sizeof(edge_rec) * (size_t)h->nf);
  if (!h->fptr || !h->fnbr || !h->fbf || !h->farea || !h->fnrm || !h->fdist || !h->vol || !cen || !er)
    FAIL(h, NBR_E_ALLOC, "alloc");
  for (int c = 0; c <= na; ++c) h->fptr[c] = cell_ptr[c];
  for (int c = 0; c < na; ++c) {
    int p0 = cell_ptr[c], np = cell_ptr[c + 1] - p0;
    if (np < 3) FAIL(h, NBR_E_INVALID, "cell %d has fewer than 3 nodes", c);
    /* shoelace area and polygon centroid */
    double A2 = 0, cx = 0, cy = 0;
    for (int k = 0; k < np; ++k) {
      int n0 = cell_nodes[p0 + k], n1 = cell_nodes[p0 + (k + 1) % np];
      if (n0 < 0 || n0 >= n_nodes || n1 < 0 || n1 >= n_nodes) FAIL(h, NBR_E_INVALID, "cell %d: bad node id", c);
      double x0 = xy[2 * n0], y0 = xy[2 * n0 + 1], x1 = xy[2 * n1], y1 = xy[2 * n1 + 1];
      double cr = x0 * y1 - x1 * y0;
      A2 += cr;
      cx += (x0 + x1) * cr;
      cy += (y0 + y1) * cr;
    }
    if (!(A2 > 0)) FAIL(h, NBR_E_INVALID, "cell %d is not counter-clockwise (area %g)", c, 0.5 * A2);
    h->vol[c] = 0.5 * A2; /* unit depth */
    cen[2 * c] = cx / (3.0 * A2);
    cen[2 * c + 1] = cy / (3.0 * A2);
    for (int k = 0; k < np; ++k) {
      int f = p0 + k, n0 = cell_nodes[p0 + k], n1 = cell_nodes[p0 + (k + 1) % np];
      double ex = xy[2 * n1] - xy[2 * n0], ey = xy[2 * n1 + 1] - xy[2 * n0 + 1];
      double len = sqrt(ex * ex + ey * ey);
      h->farea[f] = len;
      h->fnrm[3 * f] = ey / len; /* outward normal of a CCW polygon edge */
      h->fnrm[3 * f + 1] = -ex / len;
      h->fnbr[f] = -1;
      h->fbf[f] = -1;
      /* perpendicular distance centroid -> edge line (replaced for interior faces) */
      h->fdist[f] = (xy[2 * n0] - cen[2 * c]) * h->fnrm[3 * f] + (xy[2 * n0 + 1] - cen[2 * c + 1]) * h->fnrm[3 * f + 1];
      er[f].lo = n0 < n1 ? n0 : n1;
      er[f].hi = n0 < n1 ? n1 : n0;
      er[f].face = f;
    }
  }
  /* owner cell of every face index */
  int *fcell = malloc(sizeof(int) * (size_t)h->nf);
  for (int c = 0; c < na; ++c)
    for (int f = h->fptr[c]; f < h->fptr[c + 1]; ++f) fcell[f] = c;
  qsort(er, h->nf, sizeof(edge_rec), edge_cmp);
  for (int k = 0; k + 1 < h->nf; ++k) {
    if (er[k].lo == er[k + 1].lo && er[k].hi == er[k + 1].hi) {
      if (k + 2 < h->nf && er[k + 2].lo == er[k].lo && er[k + 2].hi == er[k].hi)
        FAIL(h, NBR_E_INVALID, "edge (%d,%d) is shared by more than two cells", er[k].lo, er[k].hi);
      int f0 = er[k].face, f1 = er[k + 1].face, c0 = fcell[f0], c1 = fcell[f1];
      h->fnbr[f0] = c1;
      h->fnbr[f1] = c0;
      double dx = cen[2 * c1] - cen[2 * c0], dy = cen[2 * c1 + 1] - cen[2 * c0 + 1];
      h->fdist[f0] = h->fdist[f1] = sqrt(dx * dx + dy * dy);
      ++k;
    }
  }
  int rc = copy_bf_meta(h, n_bf, bf_tag, bf_p);
  if (rc) FAIL(h, rc, "alloc");
  for (int bf = 0; bf < n_bf; ++bf) {
    int n0 = bf_nodes[2 * bf], n1 = bf_nodes[2 * bf + 1];
    edge_rec key = {n0 < n1 ? n0 : n1, n0 < n1 ? n1 : n0, -1};
    /* binary search for the first record with this (lo,hi) */
    int lo = 0, hi = h->nf;
    while (lo < hi) {
      int mid = (lo + hi) / 2;
      if (edge_cmp(&er[mid], &key) < 0) lo = mid + 1; else hi = mid;
    }
    if (lo >= h->nf || er[lo].lo != key.lo || er[lo].hi != key.hi) FAIL(h, NBR_E_INVALID, "boundary face %d: no such edge", bf);
    int f = er[lo].face;
    if (h->fnbr[f] >= 0) FAIL(h, NBR_E_INVALID, "boundary face %d is an interior edge", bf);
    if (h->fbf[f] >= 0) FAIL(h, NBR_E_INVALID, "boundary face %d listed twice", bf);
    h->fbf[f] = bf;
    h->bf_act[bf] = fcell[f];
    h->bf_face[bf] = f;
  }
  free(er);
  free(fcell);
  free(cen);
  return finish_setup(h, B, C, v, tau, share, D, s, w, n_tags, tag_type, tag_T, Qdot, T_ref, T_init, cg_rtol,
                      cg_max_iter);
}

void nanobte_ref_destroy(nanobte_ref *h) {
  if (!h) return;
  free(h->act2cell); free(h->cell2act); free(h->fptr); free(h->fnbr); free(h->fbf); free(h->farea);
  free(h->fnrm); free(h->fdist); free(h->vol); free(h->C); free(h->v); free(h->tau); free(h->share);
  free(h->s); free(h->w); free(h->bf_tag); free(h->bf_act); free(h->bf_face); free(h->bf_mirror);
  free(h->bf_p); free(h->bf_den); free(h->tag_type); free(h->tag_T); free(h->order); free(h->Qdot);
  free(h->theta); free(h->theta_prev); free(h->theta_SI); free(h->theta_en); free(h->q); free(h->eps);
  free(h->G); free(h->bcv); free(h->hist_dT); free(h->hist_cg);
  free(h);
}

int nanobte_ref_set_threads(nanobte_ref *h, int n) {
#ifdef _OPENMP
  if (n > 0) h->n_threads = n;
#else
  (void)n;
  h->n_threads = 1;
#endif
  return h->n_threads;
}

/* ------------------------------------------------------------------------------------------ */
/* O3 + O2: one transport sweep                                                                 */
/* ------------------------------------------------------------------------------------------ */
int nanobte_ref_sweep(nanobte_ref *h) {
  const int B = h->B, D = h->D, na = h->n_act;
  /* O3: boundary values from the previous iterate eps^n (lagged, R9) */
  for (int bf = 0; bf < h->n_bf; ++bf) {
    const int a = h->bf_act[bf], tag = h->bf_tag[bf], type = h->tag_type[tag];
    const double *n = h->fnrm + 3 * h->bf_face[bf];
    const double p = h->bf_p[bf];
    for (int b = 0; b < B; ++b) {
      const double Gbf = h->G[(size_t)bf * B + b];
      for (int i = 0; i < D; ++i) {
        double val = 0.0;
        if (dot3(h->s + 3 * i, n) < 0) { /* incoming direction */
          if (type == 0) {
            val = h->C[b] * (h->tag_T[tag] - h->T_ref) / h->W; /* R6 */
          } else if (type == 1) {
            val = Gbf; /* R7 */
          } else {
            int j = h->bf_mirror[(size_t)bf * D + i];
            double spec = h->eps[((size_t)b * D + j) * na + a];
            val = (type == 2) ? spec : p * spec + (1.0 - p) * Gbf; /* R8 */
          }
        }
        h->bcv[((size_t)bf * B + b) * D + i] = val;
      }
    }
  }
  /* O2: every (b, i) independently; OpenMP over directions (the paper's task parallelism) */
  int alloc_fail = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(h->n_threads)
  for (int i = 0; i < D; ++i) {
    double *g = malloc(sizeof(double) * (size_t)h->nf);
    if (!g) {
      alloc_fail = 1;
      continue;
    }
    const double *si = h->s + 3 * i;
    const int *ord = h->order + (size_t)i * na;
    /* O1: g_cf = A_cf (s_i . n_cf) / V_c */
    for (int a = 0; a < na; ++a)
      for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f) g[f] = h->farea[f] * dot3(si, h->fnrm + 3 * f) / h->vol[a];
    for (int b = 0; b < B; ++b) {
      double *e = h->eps + ((size_t)b * D + i) * na;
      const double Cb = h->C[b], vb = h->v[b], taub = h->tau[b], shb = h->share[b];
      for (int k = 0; k < na; ++k) {
        const int a = ord[k];
        double num = Cb * h->theta[a] / (h->W * taub) + h->Qdot[a] * shb / h->W; /* Eq. 11 + PAPER.md:178 */
        double den = 1.0 / taub;
        for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f) {
          if (g[f] > 0) {
            den += vb * g[f];
          } else if (g[f] < 0) {
            double up = (h->fnbr[f] >= 0) ? e[h->fnbr[f]] : h->bcv[((size_t)h->fbf[f] * B + b) * D + i];
            num += vb * (-g[f]) * up;
          }
        }
        e[a] = num / den;
      }
    }
    free(g);
  }
  if (alloc_fail) FAIL(h, NBR_E_ALLOC, "alloc in sweep");
  return NBR_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* O4 + O5: moments, diffuse averages, plain temperature update                                 */
/* ------------------------------------------------------------------------------------------ */
int nanobte_ref_update_temperature(nanobte_ref *h, double *max_dT) {
  const int B = h->B, D = h->D, na = h->n_act;
#pragma omp parallel for schedule(static) num_threads(h->n_threads)
  for (int a = 0; a < na; ++a) {
    double A1 = 0.0, A2 = 0.0, q[3] = {0, 0, 0};
    for (int b = 0; b < B; ++b) {
      double E = 0.0, F[3] = {0, 0, 0};
      for (int i = 0; i < D; ++i) {
        const double e = h->eps[((size_t)b * D + i) * na + a];
        E += h->w[i] * e;
        for (int k = 0; k < 3; ++k) F[k] += h->w[i] * h->s[3 * i + k] * e;
      }
      A1 += E / h->tau[b];
      A2 += E;
      for (int k = 0; k < 3; ++k) q[k] += h->v[b] * F[k]; /* Eq. 7 */
    }
    h->theta_SI[a] = A1 / h->beta;  /* Eq. 5 */
    h->theta_en[a] = A2 / h->Csum;  /* R13 */
    for (int k = 0; k < 3; ++k) h->q[3 * (size_t)a + k] = q[k];
  }
  /* diffuse averages for the next sweep (R7) */
  for (int bf = 0; bf < h->n_bf; ++bf) {
    const int a = h->bf_act[bf];
    const double *n = h->fnrm + 3 * h->bf_face[bf];
    for (int b = 0; b < B; ++b) {
      double num = 0.0;
      for (int i = 0; i < D; ++i) {
        double sn = dot3(h->s + 3 * i, n);
        if (sn > 0) num += h->w[i] * sn * h->eps[((size_t)b * D + i) * na + a];
      }
      h->G[(size_t)bf * B + b] = num / h->bf_den[bf];
    }
  }
  double m = 0.0;
  for (int a = 0; a < na; ++a) {
    h->theta_prev[a] = h->theta[a];
    h->theta[a] = h->theta_SI[a]; /* Eq. 6 */
    double d = fabs(h->theta[a] - h->theta_prev[a]);
    if (!(d <= m)) m = d; /* also propagates NaN */
  }
  if (max_dT) *max_dT = m;
  return isfinite(m) ? NBR_OK : NBR_E_NONFINITE;
}

/* ------------------------------------------------------------------------------------------ */
/* O6: synthetic diffusion correction                                                           */
/* ------------------------------------------------------------------------------------------ */
static void diffusion_apply(const nanobte_ref *h, const double *x, double *y) {
  for (int a = 0; a < h->n_act; ++a) {
    double acc = 0.0;
    for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f) {
      if (h->fnbr[f] >= 0)
        acc += h->kappa * h->farea[f] * (x[a] - x[h->fnbr[f]]) / h->fdist[f];
      else if (h->tag_type[h->bf_tag[h->fbf[f]]] == 0)
        acc += h->kappa * h->farea[f] * x[a] / h->fdist[f]; /* delta = 0 on the thermalizing wall */
      /* reflecting faces: zero flux */
    }
    y[a] = acc;
  }
}

int nanobte_ref_diffusion_correct(nanobte_ref *h, int *cg_iters, double *max_dT) {
  const int na = h->n_act;
  int any_therm = 0;
  for (int bf = 0; bf < h->n_bf; ++bf)
    if (h->tag_type[h->bf_tag[bf]] == 0) any_therm = 1;
  if (!any_therm) FAIL(h, NBR_E_SINGULAR, "synthetic mode needs at least one thermalizing face");
  double *rhs = malloc(sizeof(double) * na), *x = calloc(na, sizeof(double)), *r = malloc(sizeof(double) * na);
  double *p = malloc(sizeof(double) * na), *Ap = malloc(sizeof(double) * na);
  if (!rhs || !x || !r || !p || !Ap) FAIL(h, NBR_E_ALLOC, "alloc in CG");
  double bb = 0.0;
  for (int a = 0; a < na; ++a) {
    rhs[a] = h->vol[a] * h->beta * (h->theta_SI[a] - h->theta_prev[a]); /* R14c: = V (Qdot - div q^{n+1}) */
  }
  /* R14c': the face assembly of div q carries ZERO flux through reflecting walls.  The
   * cell identity above still contains the flux A_f F_f that leaked through each diffuse / specular /
   * mixed face because its incoming values lag one iteration (R9); take it out again (O8 face flux
   * with the boundary values the last sweep used).  It vanishes at convergence. */
  for (int bf = 0; bf < h->n_bf; ++bf) {
    if (h->tag_type[h->bf_tag[bf]] == 0) continue;
    const int a = h->bf_act[bf], f = h->bf_face[bf];
    const double *n = h->fnrm + 3 * f;
    double F = 0.0;
    for (int b = 0; b < h->B; ++b) {
      double Fb = 0.0;
      for (int i = 0; i < h->D; ++i) {
        double sn = dot3(h->s + 3 * i, n);
        double ef = sn > 0 ? h->eps[((size_t)b * h->D + i) * na + a] : h->bcv[((size_t)bf * h->B + b) * h->D + i];
        Fb += h->w[i] * sn * ef;
      }
      F += h->v[b] * Fb;
    }
    rhs[a] += h->farea[f] * F;
  }
  for (int a = 0; a < na; ++a) {
    r[a] = p[a] = rhs[a];
    bb += rhs[a] * rhs[a];
  }
  int it = 0;
  double rr = bb;
  const double stop2 = h->cg_rtol * h->cg_rtol * bb;
  while (rr > stop2 && it < h->cg_max_iter) {
    diffusion_apply(h, p, Ap);
    double pAp = 0.0;
    for (int a = 0; a < na; ++a) pAp += p[a] * Ap[a];
    double alpha = rr / pAp;
    double rr_new = 0.0;
    for (int a = 0; a < na; ++a) {
      x[a] += alpha * p[a];
      r[a] -= alpha * Ap[a];
      rr_new += r[a] * r[a];
    }
    double bet = rr_new / rr;
    for (int a = 0; a < na; ++a) p[a] = r[a] + bet * p[a];
    rr = rr_new;
    ++it;
  }
  double m = 0.0;
  for (int a = 0; a < na; ++a) {
    h->theta[a] = h->theta_SI[a] + x[a]; /* R14a */
    double d = fabs(h->theta[a] - h->theta_prev[a]);
    if (!(d <= m)) m = d;
  }
  free(rhs); free(x); free(r); free(p); free(Ap);
  if (cg_iters) *cg_iters = it;
  if (max_dT) *max_dT = m;
  return isfinite(m) ? NBR_OK : NBR_E_NONFINITE;
}

/* ------------------------------------------------------------------------------------------ */
/* O9: Fourier initial guess                                                                     */
/* ------------------------------------------------------------------------------------------ */
/* PAPER.md:228 (section IV): "A Fourier diffusion solve provides the initial temperature guess".  Reading R21: theta^0
 * solves the steady heat-conduction problem  -div(kappa grad theta) = Qdot  with theta = T_w - T_ref on thermalizing
 * faces and zero flux through every other boundary face, discretised with the same two-point-flux operator as the
 * synthetic correction (diffusion_apply, R14d-e: kappa from the discrete quadrature, wall distance = cell centre to face):
 *     sum_{f interior} kappa A_f (theta_c - theta_N)/d_f + sum_{f thermalizing} kappa A_f (theta_c - theta_w,f)/d_cf = V_c Qdot_c
 * solved by the same unpreconditioned CG from zero to ||r|| <= cg_rtol ||rhs||.  The distribution is not touched
 * (eps^0 stays what it is, R12); only theta is set. */
int nanobte_ref_init_fourier(nanobte_ref *h, int *cg_iters) {
  const int na = h->n_act;
  int any_therm = 0;
  for (int bf = 0; bf < h->n_bf; ++bf)
    if (h->tag_type[h->bf_tag[bf]] == 0) any_therm = 1;
  if (!any_therm) FAIL(h, NBR_E_SINGULAR, "the Fourier guess needs at least one thermalizing face");
  double *rhs = malloc(sizeof(double) * na), *x = calloc(na, sizeof(double)), *r = malloc(sizeof(double) * na);
  double *p = malloc(sizeof(double) * na), *Ap = malloc(sizeof(double) * na);
  if (!rhs || !x || !r || !p || !Ap) FAIL(h, NBR_E_ALLOC, "alloc in CG");
  for (int a = 0; a < na; ++a) {
    double acc = h->vol[a] * h->Qdot[a];
    for (int f = h->fptr[a]; f < h->fptr[a + 1]; ++f)
      if (h->fnbr[f] < 0 && h->tag_type[h->bf_tag[h->fbf[f]]] == 0)
        acc += h->kappa * h->farea[f] * (h->tag_T[h->bf_tag[h->fbf[f]]] - h->T_ref) / h->fdist[f];
    rhs[a] = acc;
  }
  double bb = 0.0;
  for (int a = 0; a < na; ++a) {
    r[a] = p[a] = rhs[a];
    bb += rhs[a] * rhs[a];
  }
  int it = 0;
  double rr = bb;
  const double stop2 = h->cg_rtol * h->cg_rtol * bb;
  while (rr > stop2 && it < h->cg_max_iter) {
    diffusion_apply(h, p, Ap);
    double pAp = 0.0;
    for (int a = 0; a < na; ++a) pAp += p[a] * Ap[a];
    double alpha = rr / pAp;
    double rr_new = 0.0;
    for (int a = 0; a < na; ++a) {
      x[a] += alpha * p[a];
      r[a] -= alpha * Ap[a];
      rr_new += r[a] * r[a];
    }
    double bet = rr_new / rr;
    for (int a = 0; a < na; ++a) p[a] = r[a] + bet * p[a];
    rr = rr_new;
    ++it;
  }
  int ok = 1;
  for (int a = 0; a < na; ++a) {
    h->theta[a] = x[a];
    ok &= isfinite(x[a]) != 0;
  }
  free(rhs); free(x); free(r); free(p); free(Ap);
  if (cg_iters) *cg_iters = it;
  return ok ? NBR_OK : NBR_E_NONFINITE;
}

/* ------------------------------------------------------------------------------------------ */
/* O7: outer loop                                                                               */
/* ------------------------------------------------------------------------------------------ */
static int push_history(nanobte_ref *h, double dT, int cg) {
  if (h->n_hist == h->cap_hist) {
    int cap = h->cap_hist ? 2 * h->cap_hist : 256;
    double *a = realloc(h->hist_dT, sizeof(double) * cap);
    int *b = realloc(h->hist_cg, sizeof(int) * cap);
    if (!a || !b) return NBR_E_ALLOC;
    h->hist_dT = a; h->hist_cg = b; h->cap_hist = cap;
  }
  h->hist_dT[h->n_hist] = dT;
  h->hist_cg[h->n_hist] = cg;
  h->n_hist++;
  return NBR_OK;
}

int nanobte_ref_solve(nanobte_ref *h, double tol, int max_iter, int mode, int *iters_out, double *last_dT_out) {
  if (mode != 0 && mode != 1) FAIL(h, NBR_E_INVALID, "mode must be 0 (plain) or 1 (synthetic)");
  h->n_hist = 0;
  double dT = INFINITY;
  int n = 0, rc = NBR_NOT_CONVERGED;
  while (n < max_iter) {
    int cg = 0, r;
    if ((r = nanobte_ref_sweep(h)) < 0) return r;
    if ((r = nanobte_ref_update_temperature(h, &dT)) < 0) return r;
    if (mode == 1 && (r = nanobte_ref_diffusion_correct(h, &cg, &dT)) < 0) return r;
    ++n;
    if ((r = push_history(h, dT, cg)) < 0) return r;
    if (dT < tol) {
      rc = NBR_OK;
      break;
    }
  }
  if (iters_out) *iters_out = n;
  if (last_dT_out) *last_dT_out = dT;
  return rc;
}

/* ------------------------------------------------------------------------------------------ */
/* getters / setters                                                                            */
/* ------------------------------------------------------------------------------------------ */
int nanobte_ref_set_T(nanobte_ref *h, const double *T) {
  for (int a = 0; a < h->n_act; ++a) h->theta[a] = T[h->act2cell[a]] - h->T_ref;
  return NBR_OK;
}

int nanobte_ref_get_T(nanobte_ref *h, int which, double *dst) {
  const double *src = which == 0 ? h->theta : which == 1 ? h->theta_en : which == 2 ? h->theta_SI : NULL;
  if (!src) FAIL(h, NBR_E_INVALID, "which must be 0, 1 or 2");
  for (int c = 0; c < h->n_cells; ++c) dst[c] = h->T_ref + (h->cell2act[c] >= 0 ? src[h->cell2act[c]] : 0.0);
  return NBR_OK;
}

int nanobte_ref_get_q(nanobte_ref *h, double *dst) {
  for (int c = 0; c < h->n_cells; ++c)
    for (int k = 0; k < h->dim; ++k) dst[(size_t)c * h->dim + k] = h->cell2act[c] >= 0 ? h->q[3 * (size_t)h->cell2act[c] + k] : 0.0;
  return NBR_OK;
}

int nanobte_ref_get_e(nanobte_ref *h, int b0, int nb, int d0, int nd, double *dst, int deviational) {
  if (b0 < 0 || nb < 0 || b0 + nb > h->B || d0 < 0 || nd < 0 || d0 + nd > h->D) FAIL(h, NBR_E_INVALID, "band/direction range");
  for (int b = 0; b < nb; ++b)
    for (int d = 0; d < nd; ++d) {
      const double *e = h->eps + ((size_t)(b0 + b) * h->D + (d0 + d)) * h->n_act;
      double *o = dst + ((size_t)b * nd + d) * h->n_cells;
      const double off = deviational ? 0.0 : h->C[b0 + b] * h->T_ref / h->W;
      for (int c = 0; c < h->n_cells; ++c) o[c] = h->cell2act[c] >= 0 ? e[h->cell2act[c]] + off : 0.0;
    }
  return NBR_OK;
}

int nanobte_ref_get_G(nanobte_ref *h, double *dst) {
  memcpy(dst, h->G, sizeof(double) * (size_t)h->n_bf * h->B);
  return NBR_OK;
}

int nanobte_ref_get_boundary_values(nanobte_ref *h, double *dst) {
  memcpy(dst, h->bcv, sizeof(double) * (size_t)h->n_bf * h->B * h->D);
  return NBR_OK;
}

/* O8: heat leaving through the boundary faces of each tag, F_f = sum_b v_b sum_i w_i (s_i.n) eps_face */
int nanobte_ref_get_boundary_heat(nanobte_ref *h, double *per_tag) {
  const int B = h->B, D = h->D, na = h->n_act;
  for (int t = 0; t < h->n_tags; ++t) per_tag[t] = 0.0;
  for (int bf = 0; bf < h->n_bf; ++bf) {
    const int a = h->bf_act[bf], f = h->bf_face[bf];
    const double *n = h->fnrm + 3 * f;
    double F = 0.0;
    for (int b = 0; b < B; ++b) {
      double Fb = 0.0;
      for (int i = 0; i < D; ++i) {
        double sn = dot3(h->s + 3 * i, n);
        double ef = sn > 0 ? h->eps[((size_t)b * D + i) * na + a] : h->bcv[((size_t)bf * B + b) * D + i];
        Fb += h->w[i] * sn * ef;
      }
      F += h->v[b] * Fb;
    }
    per_tag[h->bf_tag[bf]] += h->farea[f] * F;
  }
  return NBR_OK;
}

int nanobte_ref_get_history(nanobte_ref *h, double *dT, int32_t *cg_iters, int cap) {
  int n = h->n_hist < cap ? h->n_hist : cap;
  for (int k = 0; k < n; ++k) {
    if (dT) dT[k] = h->hist_dT[k];
    if (cg_iters) cg_iters[k] = h->hist_cg[k];
  }
  return h->n_hist;
}

int nanobte_ref_n_cells(const nanobte_ref *h) { return h->n_cells; }
int nanobte_ref_n_active(const nanobte_ref *h) { return h->n_act; }
double nanobte_ref_kappa(const nanobte_ref *h) { return h->kappa; }
const char *nanobte_ref_last_error(const nanobte_ref *h) { return h ? h->err : "null handle"; }
