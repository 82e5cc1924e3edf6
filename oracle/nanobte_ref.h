/*
 * nanobte_ref -- CPU fp64 ORACLE for the NanoBTE source-iteration hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA library (include/nanobte.h,
 * paper_2607_03226_b200/csrc/): the two were written separately from the paper.
 *
 * What it computes (citations are /root/reference/PAPER.md line numbers; where the paper
 * is silent the reading Rn of DESIGN.md "Readings" is followed and named):
 *
 *   O1  unit advection coefficients g_{cf,i} = A_cf (s_i . n_cf) / V_c            PAPER.md:104 (K_i)
 *   O2  per (band b, direction i): first-order-upwind FV solve of Eq. 4
 *         eps_c = [ C_b th_c/(W tau_b) + S_bc + v_b sum_{in} |g| eps_up ] / [ 1/tau_b + v_b sum_{out} g ]
 *       done cell by cell in a topological ("upwind first") order -- i.e. forward substitution
 *       of (I/tau + v K_i) eps = rhs.                                              (R1, R10)
 *   O3  boundary values, lagged one iteration (R9): thermalizing C_b (T_w - T_ref)/W (R6),
 *       diffuse G_bf (R7), specular eps_{b,r_f(i),c} (mirror direction), mixed p*spec+(1-p)*G (R8)
 *   O4  moments: th_SI (Eq. 5), th_en (R13), q (Eq. 7)
 *   O5  plain source iteration th <- th_SI                                         PAPER.md:62 (Eq. 6)
 *   O6  synthetic correction: CG on the two-point-flux FV diffusion operator        PAPER.md:77-97 (R14)
 *         rhs_c = V_c beta (th_SI - th^n) + sum_{reflecting faces f of c} A_f F_f   (R14c, R14c': the face
 *         assembly of div q_nonF, has zero flux through reflecting walls)
 *   O7  stop when max |th^{n+1} - th^n| < tol                                      PAPER.md:67 (R11)
 *   O8  face fluxes / boundary heat per tag (diagnostic)
 *
 * Variables are deviational (R2): eps = e - C_b T_ref / W, th = T - T_ref.
 * Source split (R5): S_{b,i,c} = Qdot_c * share_b / W, share_b = C_b / sum C.
 *
 * Parity pins (tests/test_oracle_*.py): P1 dense brute force, P2 dense global fixed point,
 * P3 closed-form discrete slab, P4 isothermal, P5 energy balance, P6 plain == synthetic,
 * P7 radiative-slab anchors, P8 symmetry.  Converged fields of the three large workloads
 * (cube 64^3, finfet, triangles 320^2) are "parity unpinned" beyond those invariants.
 *
 * Layouts: e is [band][direction][cell]; q is [cell][dim]; structured cell id =
 * i + nx*(j + ny*k); sides 0..5 = -x,+x,-y,+y,-z,+z.  Inactive cells read T_ref / 0.
 * All pointers are host pointers, read during the call and never retained.
 * Return: 0 ok, 1 not converged (state valid), < 0 error (see NBR_E_*).
 */
#ifndef NANOBTE_REF_H
#define NANOBTE_REF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct nanobte_ref nanobte_ref;

enum {
  NBR_OK = 0,
  NBR_NOT_CONVERGED = 1,
  NBR_E_INVALID = -1,
  NBR_E_ALLOC = -2,
  NBR_E_UNTAGGED = -5,
  NBR_E_SPECULAR = -6,
  NBR_E_CYCLE = -7,
  NBR_E_QUADRATURE = -8,
  NBR_E_SINGULAR = -9,
  NBR_E_NONFINITE = -10
};

int nanobte_ref_create_structured(
    int nx, int ny, int nz, const double *hx, const double *hy, const double *hz,
    const uint8_t *active /* [nx*ny*nz] or NULL */,
    int n_bf, const int32_t *bf_cell, const uint8_t *bf_side, const int32_t *bf_tag,
    const double *bf_p /* [n_bf] or NULL */,
    int B, const double *C, const double *v, const double *tau, const double *share /* or NULL */,
    int D, const double *s /* [D][3] */, const double *w,
    int n_tags, const int32_t *tag_type, const double *tag_T,
    const double *Qdot /* [n_cells] */, double T_ref, const double *T_init /* or NULL */,
    double cg_rtol, int cg_max_iter, nanobte_ref **out);

int nanobte_ref_create_unstructured(
    int n_nodes, const double *xy /* [n_nodes][2] */, int n_cells, const int32_t *cell_ptr,
    const int32_t *cell_nodes /* CCW polygons */,
    int n_bf, const int32_t *bf_nodes /* [n_bf][2] */, const int32_t *bf_tag, const double *bf_p,
    int B, const double *C, const double *v, const double *tau, const double *share,
    int D, const double *s, const double *w,
    int n_tags, const int32_t *tag_type, const double *tag_T,
    const double *Qdot, double T_ref, const double *T_init,
    double cg_rtol, int cg_max_iter, nanobte_ref **out);

void nanobte_ref_destroy(nanobte_ref *h);
int nanobte_ref_set_threads(nanobte_ref *h, int n); /* OpenMP threads for sweep/moments; returns count in use */

int nanobte_ref_sweep(nanobte_ref *h);                                   /* O3 then O2 */
int nanobte_ref_update_temperature(nanobte_ref *h, double *max_dT);      /* O4, G refresh, O5 */
int nanobte_ref_diffusion_correct(nanobte_ref *h, int *cg_iters, double *max_dT); /* O6 */
int nanobte_ref_init_fourier(nanobte_ref *h, int *cg_iters);               /* O9: theta <- Fourier solution (R21) */
int nanobte_ref_solve(nanobte_ref *h, double tol, int max_iter, int mode /*0 plain,1 synthetic*/,
                      int *iters_out, double *last_dT_out);              /* O7 */

int nanobte_ref_set_T(nanobte_ref *h, const double *T /* [n_cells] absolute */);
int nanobte_ref_get_T(nanobte_ref *h, int which /*0 T_L, 1 T_energy, 2 T_SI*/, double *dst);
int nanobte_ref_get_q(nanobte_ref *h, double *dst /* [n_cells][dim] */);
int nanobte_ref_get_e(nanobte_ref *h, int b0, int nb, int d0, int nd, double *dst /* [nb][nd][n_cells] */,
                      int deviational);
int nanobte_ref_get_G(nanobte_ref *h, double *dst /* [n_bf][B] diffuse averages (deviational) */);
int nanobte_ref_get_boundary_values(nanobte_ref *h, double *dst /* [n_bf][B][D] values used by the last sweep; 0 for outgoing */);
int nanobte_ref_get_boundary_heat(nanobte_ref *h, double *per_tag /* [n_tags], outward + */);
int nanobte_ref_get_history(nanobte_ref *h, double *dT, int32_t *cg_iters, int cap);
int nanobte_ref_n_cells(const nanobte_ref *h);
int nanobte_ref_n_active(const nanobte_ref *h);
double nanobte_ref_kappa(const nanobte_ref *h);
const char *nanobte_ref_last_error(const nanobte_ref *h);

#ifdef __cplusplus
}
#endif
#endif
