// sweep_structured.cu -- (a2)+(a4) structured transport sweep for sm_100a.
//
// What it computes (Eq. 4, 91 Eq. 11, 104/110 transport system, 178 source split; first-order upwind R1):
//   eps_c = [ C_b th_c/(W tau_b) + S_b Qdot_c + v_b sum_{a in u,v,w} |s_a|/h_a eps_up,a ] / [ 1/tau_b + v_b sum_a |s_a|/h_a ]
// for every cell c of every (band b, direction s) system, in upwind order.
//
// B200 design: the B*D systems are independent and each is a triangular solve whose
// dependency is the hyperplane u'+v'+w' = h of the direction's octant.  Instead of one launch per hyperplane over
// all systems (a chain of ~200 dependent launches with all upwind traffic through L2), ONE launch runs the whole
// sweep: a CTA (or a thread group inside it) owns a few systems for the entire grid and walks the hyperplanes
// itself.  The wavefront state -- one value per (v', w') pencil, i.e. the previous hyperplane -- lives in shared
// memory, updated in place, so the three upwind reads never leave the SM and HBM sees exactly one coalesced
// 8-byte store per update.  Threads own pencils (lines along the sweep axis u) sorted by v'+w', which makes the
// set of active pencils of a hyperplane a contiguous thread range and the global store position
// plane_off[h] + pencil index contiguous as well.
#include <algorithm>

#include "internal.h"

__device__ __forceinline__ void group_barrier(int id, int count) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

template <int GT, int RMAX, bool UNIFORM, bool HAS_W>
__global__ void __launch_bounds__((GT * RMAX >= 8) ? 512 : 1024)
    sweep_structured_kernel(const SweepArgs a, const OctTab *__restrict__ octs, const int tpg, const int ng) {
  extern __shared__ double smem[];
  const int grp = threadIdx.x / tpg, t = threadIdx.x - grp * tpg;
  const int task = blockIdx.x;
  const OctTab T = octs[a.task_oct[task]];
  const int nu = a.nu, pitch = a.pitch, slots = a.slots;
  double *buf = smem + (size_t)grp * GT * slots;

  int sys[GT];
  bool live = false;
#pragma unroll
  for (int g = 0; g < GT; ++g) {
    sys[g] = a.task_sys[((size_t)task * ng + grp) * GT + g];
    live |= sys[g] >= 0;
  }
  if (!live) return;  // padding group of the last task: uses its own named barrier, nobody waits for it
  const double *binrow[GT];
  double *erow[GT];
  double cf[GT][UNIFORM ? 5 : 6];
#pragma unroll
  for (int g = 0; g < GT; ++g) {
    const int s = sys[g] >= 0 ? sys[g] : sys[0];  // padded entries recompute system 0 and store nothing
    binrow[g] = a.bin + a.sys_bin[s];
    erow[g] = a.e + (int64_t)s * a.e_stride;
#pragma unroll
    for (int k = 0; k < (UNIFORM ? 5 : 6); ++k) cf[g][k] = a.coef[(size_t)s * 8 + k];
  }

  uint32_t pk[RMAX];
  double rv[UNIFORM ? 1 : RMAX], rw[UNIFORM ? 1 : RMAX];
#pragma unroll
  for (int r = 0; r < RMAX; ++r) {
    const int p = t + r * tpg;
    pk[r] = p < T.n_pen ? T.pen[p] : 0xffffffffu;  // m = 65535: never in range
    if (!UNIFORM) {
      const int slot = pk[r] & 0xffff;
      rv[r] = p < T.n_pen ? T.rhv[slot % pitch] : 0.0;
      rw[r] = (p < T.n_pen && HAS_W) ? T.rhw[slot / pitch] : 0.0;
    }
  }

  for (int h = 0; h < T.H; ++h) {
    const int poff = __ldg(T.plane_off + h);
    double res[RMAX][GT];
    unsigned act = 0;
#pragma unroll
    for (int r = 0; r < RMAX; ++r) {
      const int u = h - (int)(pk[r] >> 16);
      if ((unsigned)u < (unsigned)nu) {
        const int64_t pos = poff + t + r * tpg;
        const uint32_t info = __ldg(T.cellinfo + pos);
        if (!(info & 8u)) {
          act |= 1u << r;
          const double2 tq = __ldg(T.tq + pos);
          const int slot = pk[r] & 0xffff;
          const int sv = (info & 2u) ? slot : slot - 1;
          const int sw = (!HAS_W || (info & 4u)) ? slot : slot - pitch;
          double au = 0, av = 0, aw = 0;
          if (!UNIFORM) au = T.rhu[u];
#pragma unroll
          for (int g = 0; g < GT; ++g) {
            const double *b = buf + g * slots;
            double eu = b[slot], ev = b[sv], ew = HAS_W ? b[sw] : 0.0;
            if (info & 7u) {
              int idx = info >> 4;
              if (info & 1u) eu = __ldg(binrow[g] + idx++);
              if (info & 2u) ev = __ldg(binrow[g] + idx++);
              if (HAS_W && (info & 4u)) ew = __ldg(binrow[g] + idx);
            }
            double val;
            if (UNIFORM) {
              val = cf[g][0] * tq.x + cf[g][1] * tq.y + cf[g][2] * eu + cf[g][3] * ev;
              if (HAS_W) val += cf[g][4] * ew;
            } else {
              const double gu = cf[g][3] * au, gv = cf[g][4] * rv[r], gw = HAS_W ? cf[g][5] * rw[r] : 0.0;
              const double num = cf[g][0] * tq.x + cf[g][1] * tq.y + gu * eu + gv * ev + gw * ew;
              val = num / (cf[g][2] + gu + gv + gw);
            }
            res[r][g] = val;
          }
        }
      }
    }
    group_barrier(grp + 1, tpg);  // every read of hyperplane h-1 is done
#pragma unroll
    for (int r = 0; r < RMAX; ++r) {
      if (act & (1u << r)) {
        const int64_t pos = poff + t + r * tpg;
        const int slot = pk[r] & 0xffff;
#pragma unroll
        for (int g = 0; g < GT; ++g) {
          buf[g * slots + slot] = res[r][g];
          if (sys[g] >= 0) __stcs(erow[g] + pos, res[r][g]);
        }
      }
    }
    group_barrier(grp + 1, tpg);  // hyperplane h is visible
  }
}

// ---- host side: variant table ---------------------------------------------------------------------------------------
typedef void (*sweep_fn)(const SweepArgs, const OctTab *, const int, const int);

template <int GT, int RMAX>
static sweep_fn pick_uw(bool uniform, bool has_w) {
  if (uniform) return has_w ? sweep_structured_kernel<GT, RMAX, true, true> : sweep_structured_kernel<GT, RMAX, true, false>;
  return has_w ? sweep_structured_kernel<GT, RMAX, false, true> : sweep_structured_kernel<GT, RMAX, false, false>;
}
template <int GT>
static sweep_fn pick_r(int rmax, bool uniform, bool has_w) {
  switch (rmax) {
    case 1: return pick_uw<GT, 1>(uniform, has_w);
    case 2: return pick_uw<GT, 2>(uniform, has_w);
    case 4: return pick_uw<GT, 4>(uniform, has_w);
    case 8: return pick_uw<GT, 8>(uniform, has_w);
  }
  return nullptr;
}
static sweep_fn pick(int gt, int rmax, bool uniform, bool has_w) {
  switch (gt) {
    case 1: return pick_r<1>(rmax, uniform, has_w);
    case 2: return pick_r<2>(rmax, uniform, has_w);
    case 4: return pick_r<4>(rmax, uniform, has_w);
  }
  return nullptr;
}
static int max_threads(int gt, int rmax) { return gt * rmax >= 8 ? 512 : 1024; }

// Chooses systems per thread (GT), pencils per thread (RMAX), threads per group and groups per CTA.
// want_G / want_threads / want_groups: 0 = auto.
int nb_sweep_structured_config(nanobte_solver *h, int n_pen_max, int slots, int want_G, int want_threads, int want_groups,
                               int n_sys_min_class) {
  const size_t smem_cap = 227 * 1024;
  int gt = want_G > 0 ? want_G : 2;
  if (gt != 1 && gt != 2 && gt != 4) return nb_fail(h, NANOBTE_E_INVALID, "sweep_G must be 1, 2 or 4");
  if (want_G <= 0 && n_sys_min_class < 2) gt = 1;
  while (gt > 1 && (size_t)gt * slots * 8 > smem_cap) gt >>= 1;
  if ((size_t)gt * slots * 8 > smem_cap)
    return nb_fail(h, NANOBTE_E_UNSUPPORTED, "grid cross-section of %d cells needs %zu B of shared memory per system (> %zu)",
                   slots, (size_t)slots * 8, smem_cap);
  int rmax = 0, tpg = 0;
  if (want_threads > 0) {
    tpg = (want_threads + 31) / 32 * 32;
    int r = (n_pen_max + tpg - 1) / tpg;
    rmax = r <= 1 ? 1 : r <= 2 ? 2 : r <= 4 ? 4 : r <= 8 ? 8 : 0;
    if (!rmax || tpg > max_threads(gt, rmax))
      return nb_fail(h, NANOBTE_E_INVALID, "sweep_threads=%d cannot cover %d pencils", want_threads, n_pen_max);
  } else {
    const int pref[4] = {1, 2, 4, 8};
    for (int k = 0; k < 4 && !rmax; ++k) {
      int r = pref[k];
      int tt = ((n_pen_max + r - 1) / r + 31) / 32 * 32;
      // prefer at least ~4 pencils per thread on big cross-sections (fewer, fatter threads), 1 on small ones
      if (tt <= max_threads(gt, r) && (tt <= 256 || r >= 4 || k == 3)) { rmax = r; tpg = tt; }
    }
    if (!rmax) {
      for (int k = 0; k < 4 && !rmax; ++k) {
        int r = pref[k];
        int tt = ((n_pen_max + r - 1) / r + 31) / 32 * 32;
        if (tt <= max_threads(gt, r)) { rmax = r; tpg = tt; }
      }
    }
    if (!rmax)
      return nb_fail(h, NANOBTE_E_UNSUPPORTED, "grid cross-section has %d pencils; the sweep kernel supports up to %d", n_pen_max,
                     8 * 512);
  }
  int ng = want_groups > 0 ? want_groups : 1;
  ng = std::min(ng, 15);
  while (ng > 1 && (ng * tpg > max_threads(gt, rmax) || (size_t)ng * gt * slots * 8 > smem_cap)) --ng;
  h->sweep_G = gt;
  h->sweep_rmax = rmax;
  h->sweep_threads = tpg;
  h->sweep_groups = ng;
  h->sweep_smem = (size_t)ng * gt * slots * 8;
  return 0;
}

int nb_launch_sweep_structured(nanobte_solver *h) {
  sweep_fn fn = pick(h->sweep_G, h->sweep_rmax, h->uniform, h->has_w);
  if (!fn) return nb_fail(h, NANOBTE_E_INVALID, "no sweep kernel variant for G=%d R=%d", h->sweep_G, h->sweep_rmax);
  if (!h->sweep_attr_set) {
    NB_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(h->sweep_smem, 1024)));
    h->sweep_attr_set = true;
  }
  fn<<<h->n_tasks, h->sweep_groups * h->sweep_threads, h->sweep_smem, h->stream>>>(h->sw, h->d_octs, h->sweep_threads,
                                                                                   h->sweep_groups);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}
