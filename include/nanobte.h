/*
 * nanobte.h -- C ABI of the B200-native NanoBTE hot path (arxiv/paper_2607_03226).
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers; "Rn" are the readings
 * listed in DESIGN.md where the paper is silent):
 *
 *   steady, non-gray phonon BTE under the relaxation-time approximation, energy form (PAPER.md:41-55,
 *   Eq. 1-4), linearised equilibrium e0_b = C_b T_L / W (Eq. 11), discrete ordinates
 *   (PAPER.md:51, 57), first-order-upwind finite volumes (R1).  For every (band b, direction i) the
 *   transport system (I/tau_b + v_b K_i) e = e0_b/tau_b + S_b (Eq. 13) is lower
 *   triangular in upwind order and is solved as a wavefront sweep, fused with the wall closures
 *   (thermalizing / diffuse / specular / mixed-p; R6-R9), followed by the
 *   band x direction reduction to T_L (Eq. 5), T and q (Eq. 7), wrapped in
 *   plain source iteration (Eq. 6) or the synthetic, diffusion-accelerated iteration
 *   (Eq. 8-12; R14) whose macroscopic solve is a GPU conjugate gradient.
 *
 * Conventions
 *   - everything is fp64; variables are deviational about T_ref (R2): eps = e - C_b T_ref / W.
 *   - structured cell id = i + nx*(j + ny*k); side codes 0..5 = -x,+x,-y,+y,-z,+z; nz == 1 means 2-D
 *     (unit depth, only sides 0..3, s_z ignored).
 *   - direction table s is [D][3] unit vectors, weights w [D] > 0, W = sum w (Eq. 11).
 *   - tag types: 0 thermalizing (T_wall used), 1 diffuse, 2 specular, 3 mixed (per-face p in bf_p).
 *   - canonical e export layout is [band][direction][cell] over ALL n_cells (inactive cells read 0).
 *
 * Pointers: every pointer in the create_* argument structs is a HOST pointer, read during the call and
 * never retained.  Getters take `dst_is_device`: 0 = host pointer (the call synchronises the stream),
 * 1 = device pointer (copy is enqueued on the solver's stream, no synchronisation).
 * Device memory: if options.workspace is non-NULL it must be a device allocation of at least
 * nanobte_workspace_bytes_*() bytes, 256-byte aligned, owned by the caller (e.g. a torch tensor) and
 * alive until nanobte_destroy; otherwise the library allocates with cudaMalloc and frees at destroy.
 * All kernels are enqueued on options.stream (a cudaStream_t; NULL = legacy default stream), or on a second stream of the
 * library's own that is forked from and joined back into options.stream with events inside one call (the moment combine
 * runs beside the closure kernels on the tile-dataflow path; NANOBTE_NO_AUX_STREAM=1 keeps everything on one stream): towards
 * the caller every call is ordered on options.stream.
 *
 * Errors: int return; 0 OK; NANOBTE_NOT_CONVERGED (1) = state valid, max_iter reached; < 0 error.  No
 * exceptions cross the ABI, no global state; nanobte_last_error(h) gives the message.  There is NO CPU
 * fallback: without a CUDA device of compute capability 10.x every create_* fails with NANOBTE_E_ARCH.
 * A solver handle is not thread-safe.
 *
 * NANOBTE_E_SPECULAR is also returned when a direction and its mirror image carry different weights: the face
 * flux of reflecting walls is evaluated in closed form and relies on that symmetry.
 *
 * Environment hooks, read at create, for tests and tuning only (each selects another of the library's own CUDA
 * paths; none of them leaves the GPU): NANOBTE_NO_BRICK=1 (hyperplane sweep + separate moment pass instead of the
 * tile-dataflow sweep on uniform 3-D grids), NANOBTE_BRICK_SLOW_INFLOW=1 (general closure kernel of that path),
 * NANOBTE_BRICK_ENDSEG=n (planes in the end segments of long pencils on that path; 0 = even segments),
 * NANOBTE_CG_NO_MG=1 (plain fused CG instead of the multigrid-preconditioned one), NANOBTE_CG_GENERIC=1 (multi-pass
 * CG kernel), NANOBTE_CG_NO_UNI=1 (per-cell CG stencil on uniform grids; implies NO_MG), NANOBTE_CG_NO_RECYCLE=1 (plain CG
 * from zero instead of the recycled initial guess; implies NO_MG: the oracle's iterate sequence), NANOBTE_UNS_PLAIN=1
 * (non-staged unstructured sweep), NANOBTE_SWEEP_RP=0 (run-time row pitch in the hyperplane sweep), NANOBTE_CG_NBLK=k
 * (at most k CTAs in the CG kernels: more cells per thread on small meshes), NANOBTE_MG_OMEGA / NANOBTE_MG_OMEGA2 /
 * NANOBTE_MG_TAU (weights of the two Jacobi steps and over-correction of the multigrid preconditioner; defaults 1.45, 0.65
 * and 1.9; OMEGA alone sets both weights).
 */
#ifndef NANOBTE_H
#define NANOBTE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct nanobte_solver nanobte_solver;

enum {
  NANOBTE_OK = 0,
  NANOBTE_NOT_CONVERGED = 1,
  NANOBTE_E_INVALID = -1,      /* bad argument (message says which)                               */
  NANOBTE_E_ALLOC = -2,        /* host or device allocation failed / workspace too small          */
  NANOBTE_E_CUDA = -3,         /* a CUDA runtime call failed (message carries cudaGetErrorString) */
  NANOBTE_E_ARCH = -4,         /* no CUDA device, or device is not sm_100                          */
  NANOBTE_E_UNTAGGED = -5,     /* an exposed face of an active cell has no boundary tag           */
  NANOBTE_E_SPECULAR = -6,     /* mirror image of an incoming direction is not in the quadrature  */
  NANOBTE_E_CYCLE = -7,        /* upwind graph of a direction is cyclic (unstructured, R16)       */
  NANOBTE_E_QUADRATURE = -8,   /* non-unit direction, non-positive weight, or sum w s != 0        */
  NANOBTE_E_SINGULAR = -9,     /* synthetic mode without any thermalizing face                    */
  NANOBTE_E_NONFINITE = -10,   /* max|dT| is NaN/Inf                                              */
  NANOBTE_E_UNSUPPORTED = -11  /* problem shape outside what the kernels support (message)        */
};

enum { NANOBTE_THERMALIZING = 0, NANOBTE_DIFFUSE = 1, NANOBTE_SPECULAR = 2, NANOBTE_MIXED = 3 };
enum { NANOBTE_MODE_PLAIN = 0, NANOBTE_MODE_SYNTHETIC = 1 };

/* Band table: C_b [J/m^3K], v_b [m/s], tau_b [s]; src_share NULL -> C_b/sum C (R5). */
typedef struct {
  int32_t B;
  const double *C, *v, *tau;
  const double *src_share;
} nanobte_bands;

/* Angular quadrature. */
typedef struct {
  int32_t D;
  const double *s; /* [D][3] */
  const double *w; /* [D]    */
} nanobte_quadrature;

/* Boundary tag table entry. */
typedef struct {
  int32_t type;   /* NANOBTE_THERMALIZING ... NANOBTE_MIXED */
  double T_wall;  /* thermalizing only */
} nanobte_tag;

/* Structured (optionally masked) grid. */
typedef struct {
  int32_t nx, ny, nz;
  const double *hx, *hy, *hz;   /* [nx], [ny], [nz] cell sizes in metres (hz unused when nz == 1) */
  const uint8_t *active;        /* [nx*ny*nz] or NULL = all active */
  int32_t n_bfaces;
  const int32_t *bf_cell;       /* [n_bfaces] owner cell id        */
  const uint8_t *bf_side;       /* [n_bfaces] side code 0..5       */
  const int32_t *bf_tag;        /* [n_bfaces] index into tags      */
  const double *bf_p;           /* [n_bfaces] specularity of mixed faces, or NULL */
} nanobte_structured_mesh;

/* Unstructured 2-D polygon mesh (counter-clockwise cells, CSR). */
typedef struct {
  int32_t n_nodes, n_cells;
  const double *xy;             /* [n_nodes][2] */
  const int32_t *cell_ptr;      /* [n_cells+1]  */
  const int32_t *cell_nodes;    /* [cell_ptr[n_cells]] */
  int32_t n_bfaces;
  const int32_t *bf_nodes;      /* [n_bfaces][2] */
  const int32_t *bf_tag;
  const double *bf_p;
} nanobte_unstructured_mesh;

typedef struct {
  double T_ref;                 /* reference temperature of the deviational variables (R2)        */
  const double *T_init;         /* [n_cells] host, or NULL -> T_ref (R12)                          */
  void *stream;                 /* cudaStream_t                                                    */
  void *workspace;              /* device memory or NULL                                           */
  size_t workspace_bytes;
  double cg_rtol;               /* <= 0 -> 1e-12 (R14e)                                            */
  int32_t cg_max_iter;          /* <= 0 -> 100000                                                  */
  int32_t sweep_G;              /* tuning: systems per CTA in the structured sweep (1..4); 0 = auto   */
  int32_t sweep_threads;        /* tuning: compute threads per CTA of the structured sweep (<= 480); 0 = auto */
  int32_t sweep_variant;        /* 0 = auto; 3 = hyperplane sweep, single-buffered state (any spacing); 4 = hyperplane sweep,
                                   double-buffered (uniform); 5 = tile-dataflow sweep with fused moments (3-D, uniform;
                                   what auto picks there unless sweep_G / sweep_threads are given)              */
  /* Band shards (the (direction, band) tasks are distributed, the mesh is replicated, the contributions are
   * merged by one all-reduce per iteration).  A solver created on a SUBSET of the band table takes the sums over the
   * WHOLE table here (> 0; 0 = computed from the bands given): beta = sum_b C_b/tau_b (Eq. 5), sum_b C_b (R13) and
   * kappa (R14d); bands.src_share then carries the source shares of the subset in the whole table.  Its moments are the
   * subset's terms of the global sums: nanobte_export_moments / nanobte_import_moments. */
  double beta_total, Csum_total, kappa_total;
} nanobte_options;

/* Layout / schedule facts of a created solver (for reporting and roofline arithmetic). */
typedef struct {
  int32_t dim, n_cells, n_active, B, D, n_bfaces;
  int32_t n_octants;            /* direction classes in use (structured) / D (unstructured)       */
  int32_t n_planes;             /* hyperplanes per octant (structured) / max levels per direction */
  int32_t n_tasks;              /* CTAs per sweep launch                                           */
  int32_t sweep_G, sweep_threads, sweep_rmax, pencil_axis;  /* sweep_rmax: pencils per thread, 0 for the double-buffered variant */
  int64_t n_pos;                /* e slots per (band,direction) incl. holes and padding            */
  int64_t n_inflow;             /* sum over directions of boundary-inflow values per band          */
  size_t device_bytes;          /* total device memory in use by the solver                        */
  size_t sweep_smem_bytes;
  /* which CG kernel nanobte_diffusion_correct launches */
  int32_t cg_fused;             /* 1: one-barrier fused kernel, 0: multi-pass fallback                */
  int32_t cg_cells_per_thread;  /* fused kernel: 1, 2, 4 or 8                                      */
  int32_t cg_ctas;              /* CTAs of the cooperative launch (0 before the first fallback launch) */
  int32_t cg_face_uniform;      /* fused kernel: face-uniform stencil (uniform structured grids)   */
  int32_t cg_recycle;           /* fused kernel: recycled initial guess on                         */
  int32_t sweep_variant;        /* 3 / 4: hyperplane kernels, 5: tile-dataflow sweep with fused moments, 1: unstructured level sweep */
  int32_t cg_multigrid;         /* 1: nanobte_diffusion_correct runs the multigrid-preconditioned CG (uniform 3-D structured
                                   grids; cg_mg.cu); the cg_* fields above then describe the plain-CG plan kept as fallback */
  int32_t cg_mg_levels;         /* levels of its hierarchy (0 without it)                                             */
} nanobte_info;

/* Bytes of device workspace create_* would need for this problem (same validation as create). */
int nanobte_workspace_bytes_structured(const nanobte_structured_mesh *, const nanobte_bands *,
                                       const nanobte_quadrature *, const nanobte_tag *tags, int32_t n_tags,
                                       const nanobte_options *, size_t *bytes_out);
int nanobte_workspace_bytes_unstructured(const nanobte_unstructured_mesh *, const nanobte_bands *,
                                         const nanobte_quadrature *, const nanobte_tag *tags, int32_t n_tags,
                                         const nanobte_options *, size_t *bytes_out);

/* (a1) one-time setup: schedules, coefficients, reflection maps, boundary caches.
 * Qdot: [n_cells] W/m^3 host pointer or NULL.  On failure *out is still a valid handle
 * (if allocation of the handle itself succeeded) whose only use is nanobte_last_error / nanobte_destroy. */
int nanobte_create_structured(const nanobte_structured_mesh *, const nanobte_bands *, const nanobte_quadrature *,
                              const nanobte_tag *tags, int32_t n_tags, const double *Qdot,
                              const nanobte_options *, nanobte_solver **out);
int nanobte_create_unstructured(const nanobte_unstructured_mesh *, const nanobte_bands *,
                                const nanobte_quadrature *, const nanobte_tag *tags, int32_t n_tags,
                                const double *Qdot, const nanobte_options *, nanobte_solver **out);
void nanobte_destroy(nanobte_solver *);

/* (a2)-(a5) one transport sweep: eps <- (I/tau + vK)^-1 (e0(T)/tau + S + boundary inflow), PAPER.md:55, 104,
 * 110.  Boundary inflow values are the ones cached by the previous nanobte_update_temperature (R9: lagged);
 * before the first update they are the thermalizing constants and zero elsewhere (R12).  Asynchronous. */
int nanobte_sweep(nanobte_solver *);
/* keep != 0 (the default): nanobte_sweep leaves the distribution in device memory for nanobte_get_e.  keep == 0: on
 * grids swept by the tile-dataflow kernel nanobte_sweep keeps it on chip, exactly as the sweeps inside nanobte_step /
 * nanobte_solve do (see nanobte_step); the other sweep kernels always store it and ignore the setting. */
int nanobte_set_keep_e(nanobte_solver *, int32_t keep);

/* (a6) moments + closure refresh + plain update: T_SI (Eq. 5), T_energy (R13), q (Eq. 7), diffuse averages G
 * and the boundary inflow cache for the next sweep (R6-R8), T <- T_SI (Eq. 6).  max_dT (host pointer or
 * NULL) receives max_c |T_new - T_old|; the call synchronises the stream iff max_dT != NULL. */
int nanobte_update_temperature(nanobte_solver *, double *max_dT);

/* (a7) synthetic correction after update_temperature: CG on the two-point-flux diffusion operator,
 * T <- T_SI + delta (R14).  cg_iters/max_dT host pointers or NULL; synchronises.
 * Returns NANOBTE_NOT_CONVERGED (state valid, T updated with the last CG iterate) when the CG stopped on
 * options.cg_max_iter with ||r|| > cg_rtol ||rhs||. */
int nanobte_diffusion_correct(nanobte_solver *, int32_t *cg_iters, double *max_dT);

/* Band-sharded runs (Eq. 14), see nanobte_options.beta_total.  After nanobte_update_temperature on every
 * shard, nanobte_export_moments writes this shard's terms of the update, [n_active] T_SI - T_ref (Eq. 5), [n_active]
 * T_energy - T_ref (R13), [n_active][3] q (Eq. 7), [n_bfaces] the heat flux leaking through reflecting faces summed over the
 * shard's bands (R14c'), nanobte_moments_len doubles in all; the caller sums the buffers of all shards element-wise (one
 * all-reduce) and hands the result to nanobte_import_moments on every shard, which sets the three fields and the leak,
 * T <- T_SI (Eq. 6) and returns max|T_new - T_old| (host pointer or NULL; synchronises iff != NULL).  A synthetic
 * correction (nanobte_diffusion_correct) after the import uses the imported leak; every shard then solves the same
 * system and ends with the same T.  dst / src: device pointers if *_is_device != 0, else host. */
int nanobte_band_totals(const nanobte_bands *whole_table, const nanobte_quadrature *, int32_t dim,
                        double *out /* [3] host: beta, sum C, kappa of the whole table */);
int64_t nanobte_moments_len(const nanobte_solver *);
int nanobte_export_moments(nanobte_solver *, double *dst, int32_t dst_is_device);
int nanobte_import_moments(nanobte_solver *, const double *src, int32_t src_is_device, double *max_dT);

/* Fourier initial guess (section IV: "A Fourier diffusion solve provides the initial temperature guess";
 * reading R21): T <- the solution of the steady heat-conduction problem -div(kappa grad T) = Qdot with T = T_w on
 * thermalizing faces and zero flux through every other face, on the two-point-flux operator of the synthetic correction
 * (same kappa, same CG, same cg_rtol / cg_max_iter).  Replaces the lattice temperature only (as nanobte_set_T does); the
 * distribution and the wall caches keep their state, so call it before the first sweep.  cg_iters: host pointer or NULL;
 * synchronises.  NANOBTE_E_SINGULAR without a thermalizing face, NANOBTE_NOT_CONVERGED as nanobte_diffusion_correct. */
int nanobte_init_fourier(nanobte_solver *, int32_t *cg_iters);

/* One source iteration as nanobte_solve runs it: sweep, closures + moments + update and, in synthetic mode, the CG
 * correction.  On grids swept by the tile-dataflow kernel the sweep of a step keeps the
 * distribution on chip (the moments are reduced inside the sweep; only wall-cell values and tile faces
 * go to memory); nanobte_get_e afterwards first runs one storing sweep from the current T and wall cache, i.e. it
 * returns the distribution the NEXT iteration would compute (equal to the last one to the solve tolerance at
 * convergence).  nanobte_sweep always stores the distribution.  max_dT / cg_iters: host pointers or NULL; synchronises.
 * Return values as nanobte_diffusion_correct. */
int nanobte_step(nanobte_solver *, int32_t mode, double *max_dT, int32_t *cg_iters);

/* (a8) outer loop until max|dT| < tol or max_iter sweeps (R11).  Synchronises once per iteration
 * (one double device->host).  Starts the recycled CG guess afresh, so the result does not depend on earlier
 * calls on the handle.  NANOBTE_NOT_CONVERGED also when the last synthetic correction's CG did not converge. */
int nanobte_solve(nanobte_solver *, double tol, int32_t max_iter, int32_t mode, int32_t *iters_out,
                  double *last_dT_out);

int nanobte_set_T(nanobte_solver *, const double *T /* [n_cells] absolute */, int32_t src_is_device);
int nanobte_get_T(nanobte_solver *, int32_t which /* 0 T_L, 1 T_energy, 2 T_SI */, double *dst /* [n_cells] */,
                  int32_t dst_is_device);
int nanobte_get_q(nanobte_solver *, double *dst /* [n_cells][dim] */, int32_t dst_is_device);
/* dst [nb][nd][n_cells]; deviational != 0 -> eps, else e = eps + C_b T_ref / W. */
int nanobte_get_e(nanobte_solver *, int32_t b0, int32_t nb, int32_t d0, int32_t nd, double *dst,
                  int32_t deviational, int32_t dst_is_device);
int nanobte_get_G(nanobte_solver *, double *dst /* [n_bfaces][B] deviational diffuse averages */,
                  int32_t dst_is_device);
/* Heat leaving through the faces of each tag [W, or W/m in 2-D], outward positive (O8), for the last
 * sweep + update pair.  per_tag is a host pointer [n_tags]; synchronises. */
int nanobte_get_boundary_heat(nanobte_solver *, double *per_tag);
/* The same quantity (O8) for callers that may not allocate -- code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc: no cudaMalloc/cudaFree and no allocating library routine is called, by this
 * entry point or below it.  The faces of a tag are summed by 16 blocks whose partial sums go through a file-scope static
 * device array (csrc/noalloc.cu; 34 KiB, held by every GPU that loads the library until the process exits) and are joined
 * in a fixed order, so the result is reproducible run to run and equals nanobte_get_boundary_heat's up to the order of
 * the additions.  per_tag: [n_tags], caller-owned, a device pointer (dst_is_device = 1: nothing synchronises, the result
 * is ordered on the solver's stream) or a host pointer (0: synchronises).  The device the solver was created on must
 * be current, as for every call.  Errors: NANOBTE_E_INVALID if n_tags > NANOBTE_NOALLOC_MAX_TAGS (message in
 * nanobte_last_error; use nanobte_get_boundary_heat then) or a null argument; NANOBTE_E_CUDA as elsewhere.
 * All calls on one GPU share the static array, whatever the solver: calls that overlap on the GPU (other streams,
 * other threads' solvers) race on it; calls on one stream, or otherwise ordered, do not.  Nothing in it needs clearing
 * between calls (every entry that is read was written by the same call). */
#define NANOBTE_NOALLOC_MAX_TAGS 256
int nanobte_get_boundary_heat_noalloc(nanobte_solver *, double *per_tag, int32_t dst_is_device);
/* History of the last nanobte_solve: returns the number of iterations recorded, fills up to cap entries. */
int nanobte_get_history(nanobte_solver *, double *dT, int32_t *cg_iters, int32_t cap);
int nanobte_get_info(const nanobte_solver *, nanobte_info *out);
/* Number of kernels the library has launched on behalf of this solver since create. */
int64_t nanobte_launch_count(const nanobte_solver *);
double nanobte_kappa(const nanobte_solver *); /* kappa_bulk of R14d */

const char *nanobte_strerror(int code);
const char *nanobte_last_error(const nanobte_solver *);

#ifdef __cplusplus
}
#endif
#endif /* NANOBTE_H */
