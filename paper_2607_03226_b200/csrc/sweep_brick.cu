// sweep_brick.cu -- (a2)+(a4)+(a6) fused: tile-dataflow transport sweep with the moment reduction inside
// (SURVEY 8.f row f1).  See brick.h for the decomposition and the row spaces.
//
// Per update (Eq. 4, 91 Eq. 11, 104/110, 178; first-order upwind R1; uniform spacing):
//   eps_c = k_th th_c + k_Q Qdot_c + c_u eps_up,u + c_v eps_up,v + c_w eps_up,w          (coefficients pre-divided by
//   1/tau_b + v_b sum_a |s_a|/h_a, as in sweep_structured.cu)
// and per cell and u-plane the partial moments of the task's systems (Eq. 5, R13, Eq. 7):
//   part0 = sum w/tau eps, part1 = sum w eps, part2..4 = sum v w s eps.
#include <algorithm>

#include "brick.h"

namespace {

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int *p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned int ld_relaxed(const unsigned int *p) {
  unsigned int v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(unsigned int *p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// One lane per warp waits until task `up` has published at least `need` planes; the rest of the warp follows through
// __syncwarp (memory ordering among the participating lanes), and reads the published rows with L2 loads (ld.cg).
__device__ __forceinline__ void wait_progress(const unsigned int *prog, int up, unsigned int need) {
  if (up >= 0) {
    if ((threadIdx.x & 31) == 0) {
      while (ld_relaxed(prog + up) < need) __nanosleep(100);  // cheap polls; one acquire once the value is there
      (void)ld_acquire(prog + up);
    }
    __syncwarp();
  }
}

// Non-blocking form: true (in every lane) if the rows are already published.
__device__ __forceinline__ bool progress_ready(const unsigned int *prog, int up, unsigned int need) {
  if (up < 0) return true;
  int ok = 0;
  if ((threadIdx.x & 31) == 0) {
    ok = ld_relaxed(prog + up) >= need;
    if (ok) (void)ld_acquire(prog + up);
  }
  ok = __shfl_sync(0xffffffffu, ok, 0);
  __syncwarp();
  return ok != 0;
}

struct BrickSmem {
  double plane[kBrickCells * kBrickPitch];  // [cell][system]: eps of the previous u-plane (u-upwind values)
  double th[2][kBrickCells];                // theta of the plane's cells, two stages
  double qd[2][kBrickCells];                // Qdot
  unsigned long long flg[2][kBrickCells / 8];  // flag bytes, one 64-bit word per row of 8 cells
  double dcoef[32 * 4];                     // [nd][4]  w, w sx, w sy, w sz
  double bcoef[64 * 2];                     // [nb][2]  1/tau, v
  int task;
};

__global__ void __launch_bounds__(kBrickMaxS, 3) sweep_brick_kernel(const BrickArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  BrickSmem &sm = *reinterpret_cast<BrickSmem *>(smem_raw);
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;

  for (;;) {
    __syncthreads();  // the previous task's shared memory is dead
    if (t == 0) sm.task = (int)atomicAdd(a.ticket, 1u);
    __syncthreads();
    const int task = sm.task;
    if (task >= a.n_tasks) break;
    const BrickTask T = a.tasks[task];
    const BrickCG G = a.cgs[T.cg];
    const int S = G.S;
    const bool on = t < S;              // this thread owns system t of the group
    const int s = on ? t : 0;
    const double *th_g = a.th[G.cls] + T.pos0, *qd_g = a.qd[G.cls] + T.pos0;
    const uint8_t *flg_g = a.flg[G.cls] + T.pos0;
    double *inf = a.inf + G.inf_base;
    double *wall = a.wall + G.wall_base + (int64_t)T.wo0 * S + s;
    double *part = a.part + G.part_base + T.pos0;
    const int64_t npos = a.npos[G.cls];
    double *eout = a.e + G.e_base + (int64_t)T.pos0 * S + s;
    const double *irr = inf + (int64_t)T.ir0 * S + s;
    const double *fv = inf + (int64_t)T.fv0 * S + s, *fw = inf + (int64_t)T.fw0 * S + s;
    double *dn_fu = T.dn_fu0 >= 0 ? inf + (int64_t)T.dn_fu0 * S + s : nullptr;
    double *dn_fv = T.dn_fv0 >= 0 ? inf + (int64_t)T.dn_fv0 * S + s : nullptr;
    double *dn_fw = T.dn_fw0 >= 0 ? inf + (int64_t)T.dn_fw0 * S + s : nullptr;

    // coefficients of this thread's system; moment tables of the group
    const double *cf = a.coef + G.coef_base;
    const double k_th = cf[s * 5 + 0], k_Q = cf[s * 5 + 1], c_u = cf[s * 5 + 2], c_v = cf[s * 5 + 3], c_w = cf[s * 5 + 4];
    for (int k = t; k < G.nd * 4; k += kBrickMaxS) sm.dcoef[k] = cf[S * 5 + k];
    for (int k = t; k < G.nb * 2; k += kBrickMaxS) sm.bcoef[k] = cf[S * 5 + G.nd * 4 + k];

    // stage the cell tables of a plane: theta 32 x 16 B, Qdot 32 x 16 B, flags 4 x 16 B
    auto stage = [&](int un, int stg) {
      const int64_t off = (int64_t)un * kBrickCells;
      if (t < 32) cp_async16(&sm.th[stg][2 * t], th_g + off + 2 * t);
      else if (t < 64) cp_async16(&sm.qd[stg][2 * (t - 32)], qd_g + off + 2 * (t - 32));
      else if (t < 68) cp_async16(reinterpret_cast<unsigned char *>(sm.flg[stg]) + 16 * (t - 64), flg_g + off + 16 * (t - 64));
    };
    stage(0, 0);
    // u-face inflow -> plane buffer (the previous segment of the pencils, or boundary values)
    wait_progress(a.prog, T.up_u, 0x7fffffffu);
    if (on) {
      const double *fu = inf + (int64_t)T.fu0 * S + s;
#pragma unroll 8
      for (int c = 0; c < kBrickCells; ++c) sm.plane[c * kBrickPitch + s] = __ldcg(fu + (int64_t)c * S);
    }
    // v- and w-face inflow of plane 0
    double ew[kBrickTile], inv[kBrickTile];
    wait_progress(a.prog, T.up_v, 1u);
    wait_progress(a.prog, T.up_w, 1u);
#pragma unroll
    for (int k = 0; k < kBrickTile; ++k) {
      inv[k] = on ? __ldcg(fv + (int64_t)k * S) : 0.0;
      ew[k] = on ? __ldcg(fw + (int64_t)k * S) : 0.0;
    }
    cp_async_wait_all();
    __syncthreads();

    int ip = 0, wp = 0;  // next row of the IRR stream / of the wall rows (same value in every thread)
    for (int u = 0; u < T.nu; ++u) {
      const int st = u & 1;
      // stage the next plane's cell tables
      if (u + 1 < T.nu) stage(u + 1, st ^ 1);
      // ------------------------------------------ substitution: thread = system ------------------------------------------
      if (on) {
        const bool last_u = u + 1 == T.nu;
        const unsigned long long full_act = 0x0101010101010101ull >> (8 * (kBrickTile - T.tv));
        double *pl = sm.plane + s;
        for (int w = 0; w < T.tw; ++w) {
          const unsigned long long frow = sm.flg[st][w];
          double ev = inv[0];
#pragma unroll
          for (int k = 0; k + 1 < kBrickTile; ++k) inv[k] = inv[k + 1];  // inv[0] is always the current row's v-face value
          if (frow == 0ull) continue;
          const int c0 = w * kBrickTile;
          if ((frow & 0x0f0f0f0f0f0f0f0full) == full_act) {
            // ---- plain row: all tv cells active, no wall inside the tile: straight-line code, loads first ------------------
            double eu[kBrickTile], r[kBrickTile];
#pragma unroll
            for (int v = 0; v < kBrickTile; ++v) eu[v] = v < T.tv ? pl[(c0 + v) * kBrickPitch] : 0.0;
#pragma unroll
            for (int v = 0; v < kBrickTile; v += 2) {
              const double2 th2 = *reinterpret_cast<const double2 *>(&sm.th[st][c0 + v]);
              r[v] = k_th * th2.x;
              r[v + 1] = k_th * th2.y;
            }
            if (frow & 0x1010101010101010ull) {  // a source cell in the row (Qdot = 0 elsewhere)
#pragma unroll
              for (int v = 0; v < kBrickTile; v += 2) {
                const double2 q2 = *reinterpret_cast<const double2 *>(&sm.qd[st][c0 + v]);
                r[v] = fma(k_Q, q2.x, r[v]);
                r[v + 1] = fma(k_Q, q2.y, r[v + 1]);
              }
            }
#pragma unroll
            for (int v = 0; v < kBrickTile; ++v) r[v] = fma(c_u, eu[v], fma(c_w, ew[v], r[v]));
            double elast = 0.0;
#pragma unroll
            for (int v = 0; v < kBrickTile; ++v) {
              if (v < T.tv) {
                ev = fma(c_v, ev, r[v]);  // the v-chain is the only dependency between the cells of a row
                ew[v] = ev;
                pl[(c0 + v) * kBrickPitch] = ev;
                if (v + 1 == T.tv) elast = ev;
              }
            }
            if (dn_fv) dn_fv[(int64_t)(u * kBrickTile + w) * S] = elast;
            if (w + 1 == T.tw && dn_fw) {
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if (v < T.tv) dn_fw[(int64_t)(u * kBrickTile + v) * S] = ew[v];
            }
            if (last_u && dn_fu) {
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if (v < T.tv) dn_fu[(int64_t)(c0 + v) * S] = ew[v];
            }
            if (frow & 0x2020202020202020ull) {  // cells with an outgoing boundary face: eps for the closures
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if ((frow >> (8 * v)) & BRK_WALL) wall[(int64_t)(wp++) * S] = ew[v];
            }
            if (a.store_e) {
#pragma unroll
              for (int v = 0; v < kBrickTile; ++v)
                if (v < T.tv) __stcs(eout + ((int64_t)u * kBrickCells + c0 + v) * S, ew[v]);
            }
            continue;
          }
          // ---- general row: holes and walls inside the tile (values straight from L2; rare) ----------------------------------
#pragma unroll 1
          for (int v = 0; v < T.tv; ++v) {
            const unsigned f = (unsigned)(frow >> (8 * v)) & 0xffu;
            double ewv = 0.0;
#pragma unroll
            for (int k = 0; k < kBrickTile; ++k) ewv = k == v ? ew[k] : ewv;
            if (f & BRK_ACT) {
              const int cell = c0 + v;
              double eu = pl[cell * kBrickPitch];
              if (f & BRK_INJ_U) eu = __ldcg(irr + (int64_t)(ip++) * S);
              if (f & BRK_INJ_V) ev = __ldcg(irr + (int64_t)(ip++) * S);
              if (f & BRK_INJ_W) ewv = __ldcg(irr + (int64_t)(ip++) * S);
              double r = k_th * sm.th[st][cell];
              if (f & BRK_SRC) r = fma(k_Q, sm.qd[st][cell], r);
              r = fma(c_u, eu, fma(c_w, ewv, r));
              const double e = fma(c_v, ev, r);
              pl[cell * kBrickPitch] = e;
              ev = e;
              ewv = e;
              if (v + 1 == T.tv && dn_fv) dn_fv[(int64_t)(u * kBrickTile + w) * S] = e;
              if (w + 1 == T.tw && dn_fw) dn_fw[(int64_t)(u * kBrickTile + v) * S] = e;
              if (last_u && dn_fu) dn_fu[(int64_t)cell * S] = e;
              if (f & BRK_WALL) wall[(int64_t)(wp++) * S] = e;
              if (a.store_e) __stcs(eout + ((int64_t)u * kBrickCells + cell) * S, e);
            }
#pragma unroll
            for (int k = 0; k < kBrickTile; ++k) ew[k] = k == v ? ewv : ew[k];
          }
        }
      }
      cp_async_wait_all();
      __syncthreads();  // plane u is complete in the plane buffer; the staged tables of plane u+1 have landed
      if (t == 0) {  // publish: every store of the CTA before the barrier is ordered before this release
        __threadfence();
        st_release(a.prog + task, u + 1 == T.nu ? 0x7fffffffu : (unsigned)(u + 1));
      }

      // next plane's tile-face inflow: issued before the reduction if the upstream tiles are already there (the loads
      // then fly during the reduction), otherwise after it
      auto load_faces = [&](int un) {
#pragma unroll
        for (int k = 0; k < kBrickTile; ++k) {
          inv[k] = on ? __ldcg(fv + (int64_t)(un * kBrickTile + k) * S) : 0.0;
          ew[k] = on ? __ldcg(fw + (int64_t)(un * kBrickTile + k) * S) : 0.0;
        }
      };
      const bool more = u + 1 < T.nu;
      bool early = false;
      if (more) {
        early = progress_ready(a.prog, T.up_v, (unsigned)(u + 2)) && progress_ready(a.prog, T.up_w, (unsigned)(u + 2));
        if (early) load_faces(u + 1);
      }
      // ------------------------------------------ moments: lane = cell, half-warps split the bands ------------------------
      {
        const int cell = wid * 16 + (lane & 15), half = lane >> 4;
        const int nb0 = (G.nb + 1) >> 1;
        const int b_lo = half ? nb0 : 0, b_hi = half ? G.nb : nb0;
        const double *row = sm.plane + cell * kBrickPitch;
        double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0, m4 = 0.0;
        const bool act = (reinterpret_cast<const unsigned char *>(sm.flg[st])[cell] & BRK_ACT) != 0;
        if (act) {
          for (int b = b_lo; b < b_hi; ++b) {
            double E = 0.0, Fx = 0.0, Fy = 0.0, Fz = 0.0;
            const double *rb = row + b * G.nd;
            for (int d = 0; d < G.nd; ++d) {
              const double e = rb[d];
              const double2 c01 = *reinterpret_cast<const double2 *>(sm.dcoef + 4 * d);
              const double2 c23 = *reinterpret_cast<const double2 *>(sm.dcoef + 4 * d + 2);
              E = fma(c01.x, e, E);
              Fx = fma(c01.y, e, Fx);
              Fy = fma(c23.x, e, Fy);
              Fz = fma(c23.y, e, Fz);
            }
            const double2 bc = *reinterpret_cast<const double2 *>(sm.bcoef + 2 * b);
            m0 = fma(bc.x, E, m0);
            m1 += E;
            m2 = fma(bc.y, Fx, m2);
            m3 = fma(bc.y, Fy, m3);
            m4 = fma(bc.y, Fz, m4);
          }
        }
        m0 += __shfl_xor_sync(0xffffffffu, m0, 16);
        m1 += __shfl_xor_sync(0xffffffffu, m1, 16);
        m2 += __shfl_xor_sync(0xffffffffu, m2, 16);
        m3 += __shfl_xor_sync(0xffffffffu, m3, 16);
        m4 += __shfl_xor_sync(0xffffffffu, m4, 16);
        if (half == 0) {
          double *p = part + (int64_t)u * kBrickCells + cell;
          p[0] = m0;
          p[npos] = m1;
          p[2 * npos] = m2;
          p[3 * npos] = m3;
          p[4 * npos] = m4;
        }
      }
      if (more && !early) {
        wait_progress(a.prog, T.up_v, (unsigned)(u + 2));
        wait_progress(a.prog, T.up_w, (unsigned)(u + 2));
        load_faces(u + 1);
      }
      __syncthreads();  // the plane buffer and stage st are free again
    }
  }
}

}  // namespace

int nb_launch_sweep_brick(nanobte_solver *h, int store_e) {
  BrickState &bs = *h->brick;
  BrickArgs a = bs.a;
  a.store_e = store_e;
  NB_CUDA(h, cudaMemsetAsync(a.ticket, 0, sizeof(unsigned int) * (size_t)(a.n_tasks + 1), h->stream));  // ticket + progress
  NB_CUDA(h, cudaFuncSetAttribute(sweep_brick_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BrickSmem)));
  sweep_brick_kernel<<<bs.grid, kBrickMaxS, sizeof(BrickSmem), h->stream>>>(a);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  bs.e_valid = store_e != 0;
  return 0;
}

size_t nb_brick_smem_bytes() { return sizeof(BrickSmem); }
