// sweep_structured.cu -- (a2)+(a4) structured transport sweep for sm_100a.
//
// What it computes (Eq. 4, 91 Eq. 11, 104/110 transport system, 178 source split; first-order upwind R1):
//   eps_c = [ C_b th_c/(W tau_b) + S_b Qdot_c + v_b sum_{a in u,v,w} |s_a|/h_a eps_up,a ] / [ 1/tau_b + v_b sum_a |s_a|/h_a ]
// for every cell c of every (band b, direction s) system, in upwind order.
//
// B200 design: the B*D systems are independent and each is a triangular solve whose
// dependency is the hyperplane u'+v'+w' = h of the direction's octant.  Instead of one launch per hyperplane over
// all systems (a chain of ~250 dependent launches with all upwind traffic through L2), ONE launch runs the whole
// sweep: a CTA owns G systems of one octant for the entire grid and walks the hyperplanes itself.
//   * The wavefront state -- one value per (v', w') pencil and system, i.e. the previous hyperplane -- lives in
//     shared memory, so the v/w upwind reads never leave the SM; the u upwind value is the thread's own previous
//     result and stays in a register.
//   * Threads own pencils (lines along the sweep axis u) sorted by v'+w': the active pencils of a hyperplane are a
//     contiguous slot range [lo, lo+cnt) of the state rows, and their positions in the e rows are contiguous too.
//     So the state row segment IS the output: after every hyperplane one elected thread of a dedicated DMA warp
//     issues one bulk TMA store (cp.async.bulk shared -> global) per system.  The compute warps never form a
//     global address; HBM sees exactly one 8-byte streaming write per update, in >= 128-byte aligned segments.
//   * Everything a hyperplane consumes arrives by 1-D bulk TMA two planes ahead, into a two-stage ring, on one
//     mbarrier: the per-cell tables (flags / inflow index, theta, Qdot) and, per system, the hyperplane's slice
//     of the lagged boundary-inflow cache (R9), which lands right behind the state row so that "upwind value" is
//     one shared-memory load whether it is an interior neighbour or a wall.
#include <algorithm>
#include <cstdlib>

#include "internal.h"

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// 1-D bulk TMA global -> shared, completion on an mbarrier (bytes: multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// 1-D bulk TMA shared -> global (bulk async-group completion)
__device__ __forceinline__ void tma_store_1d(void *dst, const void *src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// CTA-wide barrier that the compute warps and the DMA warp reach from different program points
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Shared-memory carve-up (all offsets multiples of 16 bytes).  A system's row is [ state sp | inflow stage 0 gcap |
// inflow stage 1 gcap ] doubles, so one index addresses "upwind value" wherever it comes from.
struct SmemLayout {
  uint32_t tq, q, rows, plane, bar, total, rp;
};
__host__ __device__ inline SmemLayout smem_layout(int G, int sp, int pcap, int gcap, int qcap, int H, int rp_fixed) {
  SmemLayout L;
  L.rp = rp_fixed ? (uint32_t)rp_fixed : (uint32_t)sp + 2u * (uint32_t)gcap;  // row pitch in doubles (even)
  L.tq = 0;                                                  // [2][pcap] double2
  L.q = L.tq + 2u * (uint32_t)pcap * 16u;                    // [2][qcap] double
  L.rows = L.q + 2u * (uint32_t)qcap * 8u;                   // [G][rp]   double
  L.plane = L.rows + (uint32_t)G * L.rp * 8u;                // [H+1][2]  int4
  L.bar = L.plane + ((uint32_t)H + 1u) * 32u;                // [2]       mbarrier
  L.total = L.bar + 16u;
  return L;
}

// blockDim.x = NT compute threads + 32 (the DMA warp).  R = pencils per compute thread.  RP > 0: the row pitch is this
// compile-time constant (>= sp + 2 gcap), so the per-system shared-memory offsets g*RP*8 fold into the LDS/STS
// instructions as immediates (27 % of the executed instructions were the IMADs that formed them); RP = 0: run-time pitch.
template <int G, int R, bool UNIFORM, int RP>
__global__ void __launch_bounds__(512) sweep_structured_kernel(const SweepArgs a, const OctTab *__restrict__ octs) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int t = threadIdx.x, nt = blockDim.x - 32;
  const int task = blockIdx.x;
  const OctTab T = octs[a.task_oct[task]];
  const int nu = a.nu, sp = a.sp, pcap = a.pcap, gcap = a.gcap, qcap = a.qcap;
  const SmemLayout L = smem_layout(G, sp, pcap, gcap, qcap, T.H, RP);
  double2 *tq_s = reinterpret_cast<double2 *>(smem + L.tq);
  double *q_s = reinterpret_cast<double *>(smem + L.q);
  double *rows = reinterpret_cast<double *>(smem + L.rows);
  int4 *plane_s = reinterpret_cast<int4 *>(smem + L.plane);
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + L.bar);
  const uint32_t rp = RP ? (uint32_t)RP : L.rp;

  const int row_loc = a.task_row[task];
  const int n_valid = min(G, T.n_rows - row_loc);  // rows past the class's end recompute the last row and store nothing
  const int64_t row_g0 = (int64_t)T.row0 + row_loc;

  for (int k = t; k < 2 * (T.H + 1); k += blockDim.x) plane_s[k] = T.plane[k];
  for (uint32_t k = t; k < (uint32_t)G * rp; k += blockDim.x) rows[k] = 0.0;
  if (t == 0) {
    mbar_init(bar, 1);
    mbar_init(bar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  fence_proxy_async();
  __syncthreads();

  if (t >= nt) {
    // ------------------------------------------------ DMA warp ---------------------------------------------------
    const bool lead = t == nt;
    double *const e0 = a.e + row_g0 * a.e_stride;
    const double *const bin0 = a.bin + T.bin_base + (int64_t)row_loc * T.n_in;
    auto issue_loads = [&](int h) {  // tables + inflow slices of hyperplane h into stage h & 1
      const int4 P = plane_s[2 * h], Q = plane_s[2 * h + 1];
      const int s = h & 1;
      const uint32_t c4 = ((uint32_t)(P.y + P.w) + 3u) & ~3u;
      const uint32_t nin = (uint32_t)(plane_s[2 * h + 3].y - Q.y);  // even
      const uint32_t nq = (uint32_t)(plane_s[2 * h + 3].z - Q.z);   // even
      mbar_expect_tx(bar + s, c4 * 16u + nq * 8u + (uint32_t)G * nin * 8u);
      if (c4) tma_load_1d(tq_s + (size_t)s * pcap, T.tq + Q.x, c4 * 16u, bar + s);
      if (nq) tma_load_1d(q_s + (size_t)s * qcap, T.qlist + Q.z, nq * 8u, bar + s);
      if (nin) {
#pragma unroll
        for (int g = 0; g < G; ++g)
          tma_load_1d(rows + (size_t)g * rp + sp + s * gcap, bin0 + (int64_t)min(g, n_valid - 1) * T.n_in + Q.y, nin * 8u, bar + s);
      }
    };
    if (lead) {
      issue_loads(0);
      if (T.H > 1) issue_loads(1);
    }
    for (int h = 0; h < T.H; ++h) {
      if (lead) tma_store_wait_read();  // the stores of hyperplane h-1 have read the state rows
      cta_sync();  // A: every read of hyperplane h-1 and of stage h&1 is done
      // two planes ahead, and ahead of this plane's stores in the TMA queue
      if (lead && h + 2 < T.H) issue_loads(h + 2);
      cta_sync();  // B: hyperplane h is in the state rows (and fenced to the async proxy)
      if (lead) {
        const int4 P = plane_s[2 * h];
        const int start = plane_s[2 * h + 1].x;
#pragma unroll
        for (int g = 0; g < G; ++g)
          if (g < n_valid) {  // the plane's wall cells, then its interior cells: two contiguous slot ranges
            if (P.y) tma_store_1d(e0 + (int64_t)g * a.e_stride + start, rows + (size_t)g * rp + P.x, (uint32_t)P.y * 8u);
            if (P.w) tma_store_1d(e0 + (int64_t)g * a.e_stride + start + P.y, rows + (size_t)g * rp + P.z, (uint32_t)P.w * 8u);
          }
        tma_store_commit();
      }
    }
    if (lead) tma_store_wait_read();
    return;
  }

  // -------------------------------------------------- compute warps ------------------------------------------------
  double cf[G][UNIFORM ? 5 : 6];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int64_t row = row_g0 + min(g, n_valid - 1);
#pragma unroll
    for (int k = 0; k < (UNIFORM ? 5 : 6); ++k) cf[g][k] = a.coef[row * 8 + k];
  }
  // per-thread pencils: slot p = t + r*nt; upwind pencil slots (the zero slot n_pen if there is none)
  int pm[UNIFORM ? 1 : R];
  double rv[UNIFORM ? 1 : R], rw[UNIFORM ? 1 : R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int p = t + r * nt;
    if (!UNIFORM) { rv[r] = rw[r] = 0.0; pm[r] = 0; }
    if (!UNIFORM && p < T.n_pen) {
      const uint2 q = T.pen[p];
      {
        pm[r] = (int)q.x;
        const double2 rh = T.pen_rh[p];
        rv[r] = rh.x;
        rw[r] = rh.y;
      }
    }
  }
  double res[R][G];
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int g = 0; g < G; ++g) res[r][g] = 0.0;

  int4 Pn = plane_s[0];
  for (int h = 0; h < T.H; ++h) {
    const int s = h & 1;
    const int4 P = Pn;  // {first wall slot, wall slots, first interior slot, interior slots} of this hyperplane
    Pn = plane_s[2 * h + 2];
    mbar_wait(bar + s, (h >> 1) & 1);
    const double2 *tqh = tq_s + (size_t)s * pcap;
    const double *qh = q_s + (size_t)s * qcap;
    const uint32_t gs = (uint32_t)sp + (uint32_t)(s * gcap);  // this hyperplane's inflow stage within a row
    unsigned act = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int p = t + r * nt;
      const unsigned kw = (unsigned)(p - P.x), ki = (unsigned)(p - P.z);
      if (kw < (unsigned)P.y || ki < (unsigned)P.w) {
        const unsigned k = kw < (unsigned)P.y ? kw : ki + (unsigned)P.y;  // index within the plane's segment
        double2 tq = tqh[k];
        const uint64_t rec = (uint64_t)__double_as_longlong(tq.y);
        const uint32_t info = (uint32_t)rec, pnb = (uint32_t)(rec >> 32);
        if (!(info & 8u)) {  // not a hole / padding slot
          act |= 1u << r;
          tq.y = (info & 16u) ? qh[info >> 18] : 0.0;  // Qdot of a source cell
          const uint32_t gb = gs + ((info >> 5) & 0x1fffu);
          const uint32_t iv = (info & 2u) ? gb + (info & 1u) : (pnb & 0xffffu);
          const uint32_t iw = (info & 4u) ? gb + (info & 1u) + ((info >> 1) & 1u) : (pnb >> 16);
          double eu[G], ev[G], ew[G];
#pragma unroll
          for (int g = 0; g < G; ++g) {
            eu[g] = res[r][g];
            ev[g] = rows[g * rp + iv];
            ew[g] = rows[g * rp + iw];
          }
          if (info & 1u) {
#pragma unroll
            for (int g = 0; g < G; ++g) eu[g] = rows[g * rp + gb];
          }
          if (UNIFORM) {
#pragma unroll
            for (int g = 0; g < G; ++g)
              res[r][g] = cf[g][0] * tq.x + cf[g][1] * tq.y + cf[g][2] * eu[g] + cf[g][3] * ev[g] + cf[g][4] * ew[g];
          } else {
            const double au = __ldg(T.rhu + min(max(h - pm[r], 0), nu - 1));
#pragma unroll
            for (int g = 0; g < G; ++g) {
              const double gu = cf[g][3] * au, gv = cf[g][4] * rv[r], gw = cf[g][5] * rw[r];
              const double num = cf[g][0] * tq.x + cf[g][1] * tq.y + gu * eu[g] + gv * ev[g] + gw * ew[g];
              res[r][g] = num / (cf[g][2] + gu + gv + gw);
            }
          }
        }
      }
    }
    cta_sync();  // A: every read of hyperplane h-1 (and of stage s) is done; its stores have left the state rows
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (act & (1u << r)) {
        const int p = t + r * nt;
#pragma unroll
        for (int g = 0; g < G; ++g) rows[g * rp + p] = res[r][g];
      }
    }
    fence_proxy_async();  // generic-proxy writes -> visible to the bulk store the DMA warp issues after B
    cta_sync();           // B: hyperplane h is visible
  }
}

// =================================================================================================================
// Double-buffered variant (uniform spacing; sweep_variant = 4, not the default: measured on B200 it halves the fixed
// per-hyperplane cost but its fourth shared-memory access per update -- the u-upwind value -- costs more than that on
// the large grids, where the shared-memory pipe is the busiest unit).  The state rows exist
// twice: hyperplane h is written to buffer h&1 while buffer (h-1)&1 is read, so
//   * there is ONE CTA barrier per hyperplane and no write phase (results go straight to shared memory),
//   * cells are assigned to threads per hyperplane (thread t takes the plane's cells t, t+nt, ...), so no
//     iteration is spent on pencils that are not active in this plane, and nothing per pencil lives in registers:
//     the u-upwind value is the pencil's own slot in the other buffer, the upwind slots come with the cell record.
// Row of a system: [ state buffer 0 | state buffer 1 | inflow stage 0 | inflow stage 1 ].
// =================================================================================================================
struct SmemLayoutDB {
  uint32_t tq, q, rows, plane, bar, total, rp;
};
__host__ __device__ inline SmemLayoutDB smem_layout_db(int G, int sp, int pcap, int gcap, int qcap, int H) {
  SmemLayoutDB L;
  L.rp = 2u * (uint32_t)sp + 2u * (uint32_t)gcap;
  L.tq = 0;                                                  // [2][pcap] double2 records
  L.q = L.tq + 2u * (uint32_t)pcap * 16u;                    // [2][qcap] double
  L.rows = L.q + 2u * (uint32_t)qcap * 8u;                   // [G][rp]   double
  L.plane = L.rows + (uint32_t)G * L.rp * 8u;                // [H+1][2]  int4
  L.bar = L.plane + ((uint32_t)H + 1u) * 32u;                // [2]       mbarrier
  L.total = L.bar + 16u;
  return L;
}

template <int G>
__global__ void __launch_bounds__(512) sweep_structured_db_kernel(const SweepArgs a, const OctTab *__restrict__ octs) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int t = threadIdx.x, nt = blockDim.x - 32;
  const int task = blockIdx.x;
  const OctTab T = octs[a.task_oct[task]];
  const int sp = a.sp, pcap = a.pcap, gcap = a.gcap, qcap = a.qcap;
  const SmemLayoutDB L = smem_layout_db(G, sp, pcap, gcap, qcap, T.H);
  double2 *tq_s = reinterpret_cast<double2 *>(smem + L.tq);
  double *q_s = reinterpret_cast<double *>(smem + L.q);
  double *rows = reinterpret_cast<double *>(smem + L.rows);
  int4 *plane_s = reinterpret_cast<int4 *>(smem + L.plane);
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + L.bar);
  const uint32_t rp = L.rp;

  const int row_loc = a.task_row[task];
  const int n_valid = min(G, T.n_rows - row_loc);
  const int64_t row_g0 = (int64_t)T.row0 + row_loc;

  for (int k = t; k < 2 * (T.H + 1); k += blockDim.x) plane_s[k] = T.plane[k];
  for (uint32_t k = t; k < (uint32_t)G * rp; k += blockDim.x) rows[k] = 0.0;
  if (t == 0) {
    mbar_init(bar, 1);
    mbar_init(bar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  fence_proxy_async();
  __syncthreads();

  if (t >= nt) {
    // ------------------------------------------------ DMA warp ---------------------------------------------------
    const bool lead = t == nt;
    double *const e0 = a.e + row_g0 * a.e_stride;
    const double *const bin0 = a.bin + T.bin_base + (int64_t)row_loc * T.n_in;
    auto issue_loads = [&](int h) {
      const int4 P = plane_s[2 * h], Q = plane_s[2 * h + 1];
      const int s = h & 1;
      const uint32_t c4 = ((uint32_t)(P.y + P.w) + 3u) & ~3u;
      const uint32_t nin = (uint32_t)(plane_s[2 * h + 3].y - Q.y);
      const uint32_t nq = (uint32_t)(plane_s[2 * h + 3].z - Q.z);
      mbar_expect_tx(bar + s, c4 * 16u + nq * 8u + (uint32_t)G * nin * 8u);
      if (c4) tma_load_1d(tq_s + (size_t)s * pcap, T.tq + Q.x, c4 * 16u, bar + s);
      if (nq) tma_load_1d(q_s + (size_t)s * qcap, T.qlist + Q.z, nq * 8u, bar + s);
      if (nin) {
#pragma unroll
        for (int g = 0; g < G; ++g)
          tma_load_1d(rows + (size_t)g * rp + 2 * sp + s * gcap, bin0 + (int64_t)min(g, n_valid - 1) * T.n_in + Q.y, nin * 8u, bar + s);
      }
    };
    if (lead) {
      issue_loads(0);
      if (T.H > 1) issue_loads(1);
    }
    for (int h = 0; h < T.H; ++h) {
      // the stores of hyperplane h-1 have read buffer (h-1)&1, which hyperplane h+1 overwrites after this barrier
      if (lead) tma_store_wait_read();
      cta_sync();  // hyperplane h is complete in buffer h&1; stage h&1 is free
      if (lead) {
        const int4 P = plane_s[2 * h];
        const int start = plane_s[2 * h + 1].x;
        const double *buf = rows + (size_t)(h & 1) * sp;
#pragma unroll
        for (int g = 0; g < G; ++g)
          if (g < n_valid) {
            if (P.y) tma_store_1d(e0 + (int64_t)g * a.e_stride + start, buf + (size_t)g * rp + P.x, (uint32_t)P.y * 8u);
            if (P.w) tma_store_1d(e0 + (int64_t)g * a.e_stride + start + P.y, buf + (size_t)g * rp + P.z, (uint32_t)P.w * 8u);
          }
        tma_store_commit();
        if (h + 2 < T.H) issue_loads(h + 2);
      }
    }
    if (lead) tma_store_wait_read();
    return;
  }

  // -------------------------------------------------- compute warps ------------------------------------------------
  double cf[G][5];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int64_t row = row_g0 + min(g, n_valid - 1);
#pragma unroll
    for (int k = 0; k < 5; ++k) cf[g][k] = a.coef[row * 8 + k];
  }
  int4 Pn = plane_s[0];
  for (int h = 0; h < T.H; ++h) {
    const int s = h & 1;
    const int4 P = Pn;
    Pn = plane_s[2 * h + 2];
    const int ntot = P.y + P.w;
    const uint32_t prev = (uint32_t)((s ^ 1) * sp), cur = (uint32_t)(s * sp);
    const uint32_t gs = 2u * (uint32_t)sp + (uint32_t)(s * gcap);
    const double2 *tqh = tq_s + (size_t)s * pcap;
    const double *qh = q_s + (size_t)s * qcap;
    mbar_wait(bar + s, (h >> 1) & 1);
    for (int k0 = t; k0 < ntot; k0 += 2 * nt) {  // two cells per trip: all shared-memory loads before the first store
      double res[2][G];
      uint32_t slot[2];
      bool on[2];
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int k = k0 + j * nt;
        on[j] = false;
        slot[j] = 0;
        if (k < ntot) {
          double2 tq = tqh[k];
          const uint64_t rec = (uint64_t)__double_as_longlong(tq.y);
          const uint32_t info = (uint32_t)rec, pnb = (uint32_t)(rec >> 32);
          if (!(info & 8u)) {
            on[j] = true;
            const uint32_t p = k < P.y ? (uint32_t)(P.x + k) : (uint32_t)(P.z + k - P.y);
            slot[j] = p;
            const double qd = (info & 16u) ? qh[info >> 18] : 0.0;
            const uint32_t gb = gs + ((info >> 5) & 0x1fffu);
            const uint32_t iu = (info & 1u) ? gb : prev + p;
            const uint32_t iv = (info & 2u) ? gb + (info & 1u) : prev + (pnb & 0xffffu);
            const uint32_t iw = (info & 4u) ? gb + (info & 1u) + ((info >> 1) & 1u) : prev + (pnb >> 16);
#pragma unroll
            for (int g = 0; g < G; ++g) {
              const double *rg = rows + g * rp;
              res[j][g] = cf[g][0] * tq.x + cf[g][1] * qd + cf[g][2] * rg[iu] + cf[g][3] * rg[iv] + cf[g][4] * rg[iw];
            }
          }
        }
      }
#pragma unroll
      for (int j = 0; j < 2; ++j)
        if (on[j]) {
#pragma unroll
          for (int g = 0; g < G; ++g) rows[g * rp + cur + slot[j]] = res[j][g];
        }
    }
    fence_proxy_async();
    cta_sync();
  }
}

// ---- host side: variant table ---------------------------------------------------------------------------------------
typedef void (*sweep_fn)(const SweepArgs, const OctTab *);
constexpr int kMaxGR = 24;  // registers: 2*G*R hold the results of a hyperplane; larger products spill

template <int G, int RP>
sweep_fn pick_r(int r, bool uniform) {
#define NB_CASE(RR)                                                                                              \
  case RR:                                                                                                       \
    if constexpr (RP == 0 && G * RR <= kMaxGR / 2) { if (!uniform) return sweep_structured_kernel<G, RR, false, 0>; } \
    if constexpr (G * RR <= kMaxGR && (RP == 0 || (G >= 2 && RR >= 4 && RR <= 6))) { if (uniform) return sweep_structured_kernel<G, RR, true, RP>; } \
    break;
  switch (r) {
    NB_CASE(1)
    NB_CASE(2)
    NB_CASE(3)
    NB_CASE(4)
    NB_CASE(5)
    NB_CASE(6)
    NB_CASE(8)
    NB_CASE(10)
    NB_CASE(12)
  }
#undef NB_CASE
  return nullptr;
}
template <int RP>
sweep_fn pick_g(int g, int r, bool uniform) {
  switch (g) {
    case 1: return pick_r<1, RP>(r, uniform);
    case 2: return pick_r<2, RP>(r, uniform);
    case 3: return pick_r<3, RP>(r, uniform);
    case 4: return pick_r<4, RP>(r, uniform);
  }
  return nullptr;
}
// compile-time row pitches on offer (doubles); a grid whose rows need more, or a small launch shape, runs with RP = 0
const int kRowPitch[4] = {2048, 3072, 4096, 5120};
sweep_fn pick(int g, int r, bool uniform, int rp) {
  switch (rp) {
    case 0: return pick_g<0>(g, r, uniform);
    case 2048: return pick_g<2048>(g, r, uniform);
    case 3072: return pick_g<3072>(g, r, uniform);
    case 4096: return pick_g<4096>(g, r, uniform);
    case 5120: return pick_g<5120>(g, r, uniform);
  }
  return nullptr;
}
const int kR[9] = {1, 2, 3, 4, 5, 6, 8, 10, 12};
const int kNR = 9;
const int kMaxCompute = 480;  // + the DMA warp = 512 threads

}  // namespace

// Chooses systems per CTA (G), pencils per thread (R) and compute threads per CTA.  want_G / want_threads: 0 = auto.
// n_pen_max: pencil slots (incl. padding); p_max: largest hyperplane; gcap: largest per-hyperplane inflow slice.
int nb_sweep_structured_config(nanobte_solver *h, int n_pen_max, int p_max, int gcap, int qcap, int H, int want_G, int want_threads,
                               int n_sys_min_class, int want_variant, int n_sys_total) {
  const size_t smem_cap = 227 * 1024;
  if (want_G < 0 || want_G > 4) return nb_fail(h, NANOBTE_E_INVALID, "sweep_G must be 0..4");
  if (n_pen_max > 12 * kMaxCompute || n_pen_max >= 65535)
    return nb_fail(h, NANOBTE_E_UNSUPPORTED, "grid cross-section has %d pencils; the sweep kernel supports up to %d", n_pen_max,
                   12 * kMaxCompute);
  int R = 0, T = 0;
  if (want_threads > 0) {
    T = std::min(kMaxCompute, (want_threads + 31) / 32 * 32);
    for (int k = 0; k < kNR && !R; ++k)
      if ((long)kR[k] * T >= n_pen_max) R = kR[k];
    if (!R) return nb_fail(h, NANOBTE_E_INVALID, "sweep_threads=%d cannot cover %d pencils", want_threads, n_pen_max);
  } else {
    for (int k = 0; k < kNR && !R; ++k) {
      const int tt = ((n_pen_max + kR[k] - 1) / kR[k] + 31) / 32 * 32;
      if (tt <= kMaxCompute) { R = kR[k]; T = tt; }
    }
    // with several pencils per thread the CTA is alone on its SM anyway: more warps hide more latency (config 3: -2 %)
    if (R >= 4) T = kMaxCompute;
  }
  const int sp = (n_pen_max + 1 + 1) & ~1;
  const int pcap = (p_max + 3 + 4) & ~3;
  gcap = (gcap + 1) & ~1;
  qcap = (qcap + 1) & ~1;
  int G = 0;
  const int cand[4] = {4, 3, 2, 1};
  for (int k = 0; k < 4 && !G; ++k) {
    const int g = cand[k];
    if (want_G > 0 && g != want_G) continue;
    if (smem_layout(g, sp, pcap, gcap, qcap, H, 0).total > smem_cap) continue;
    if (g * R > (h->uniform ? kMaxGR : kMaxGR / 2)) continue;  // the non-uniform variant carries 5 more registers per pencil
    if (want_G <= 0 && g > std::max(1, n_sys_min_class)) continue;
    // small problems: rather more CTAs than more systems per CTA, until the machine has two CTAs per SM to run
    if (want_G <= 0 && g > 1 && (long)((n_sys_total + g - 1) / g) < 2L * h->n_sm) continue;
    G = g;
  }
  if (!G) {
    if (want_G > 0) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "sweep_G=%d with %d pencils per thread needs %u B of shared memory (cap %zu) and G*R <= %d",
                                   want_G, R, smem_layout(want_G, sp, pcap, gcap, qcap, H, 0).total, smem_cap, kMaxGR);
    return nb_fail(h, NANOBTE_E_UNSUPPORTED, "grid cross-section of %d pencils needs %u B of shared memory (> %zu)", n_pen_max,
                   smem_layout(1, sp, pcap, gcap, qcap, H, 0).total, smem_cap);
  }
  // double-buffered variant: uniform spacing only, on request
  h->sweep_variant = 3;
  if (h->uniform && want_variant == 4) {
    int Gd = 0;
    for (int k = 0; k < 4 && !Gd; ++k) {
      const int g = cand[k];
      if (want_G > 0 && g != want_G) continue;
      if (smem_layout_db(g, sp, pcap, gcap, qcap, H).total > smem_cap) continue;
      if (want_G <= 0 && g > std::max(1, n_sys_min_class)) continue;
      Gd = g;
    }
    if (Gd) {
      h->sweep_variant = 4;
      h->sweep_G = Gd;
      h->sweep_rmax = 0;
      h->sweep_threads = want_threads > 0 ? T : std::min(kMaxCompute, std::max(32, (p_max / 2 + 31) / 32 * 32));
      h->sweep_smem = smem_layout_db(Gd, sp, pcap, gcap, qcap, H).total;
      h->sw.sp = sp;
      h->sw.pcap = pcap;
      h->sw.gcap = gcap;
      h->sw.qcap = qcap;
      return 0;
    }
    if (want_variant == 4) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "the double-buffered sweep does not fit in shared memory");
  } else if (want_variant == 4) {
    return nb_fail(h, NANOBTE_E_UNSUPPORTED, "the double-buffered sweep needs uniform spacing");
  }
  h->sweep_G = G;
  h->sweep_rmax = R;
  h->sweep_threads = T;
  h->sweep_rp = 0;
  const char *rp_env = std::getenv("NANOBTE_SWEEP_RP");  // tuning hook: 0 forces the run-time pitch
  // measured on B200: -6 % on config 4 (G = 4, R = 5), but +30 % with 10 pencils per thread (config 3), hence R <= 6
  if (h->uniform && G >= 2 && R >= 4 && R <= 6 && !(rp_env && std::atoi(rp_env) == 0)) {
    for (int k = 0; k < 4 && !h->sweep_rp; ++k)
      if (kRowPitch[k] >= sp + 2 * gcap && smem_layout(G, sp, pcap, gcap, qcap, H, kRowPitch[k]).total <= smem_cap) h->sweep_rp = kRowPitch[k];
  }
  h->sweep_smem = smem_layout(G, sp, pcap, gcap, qcap, H, h->sweep_rp).total;
  h->sw.sp = sp;
  h->sw.pcap = pcap;
  h->sw.gcap = gcap;
  h->sw.qcap = qcap;
  return 0;
}

int nb_launch_sweep_structured(nanobte_solver *h) {
  sweep_fn fn = nullptr;
  if (h->sweep_variant == 4) {
    switch (h->sweep_G) {
      case 1: fn = sweep_structured_db_kernel<1>; break;
      case 2: fn = sweep_structured_db_kernel<2>; break;
      case 3: fn = sweep_structured_db_kernel<3>; break;
      case 4: fn = sweep_structured_db_kernel<4>; break;
    }
  } else {
    fn = pick(h->sweep_G, h->sweep_rmax, h->uniform, h->sweep_rp);
  }
  if (!fn) return nb_fail(h, NANOBTE_E_INVALID, "no sweep kernel variant for G=%d R=%d", h->sweep_G, h->sweep_rmax);
  // the attribute belongs to the function, not to this solver: another solver that picked the same instantiation may have
  // set a smaller cap since our last launch, so it is (re)set before every launch
  NB_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(h->sweep_smem, 1024)));
  fn<<<h->n_tasks, h->sweep_threads + 32, h->sweep_smem, h->stream>>>(h->sw, h->d_octs);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}
