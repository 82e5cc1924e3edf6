// sweep_unstructured.cu -- (a1)+(a2)+(a5)+(a6) for unstructured 2-D polygon meshes (BASELINE.json configs[4]):
// one-time setup (geometry, per-direction level schedules, closure tables, diffusion stencil), the level-scheduled
// transport sweep, and the band x direction moment reduction in the per-direction layout.
//
// What the sweep computes (Eq. 4, 91 Eq. 11, 104/110 transport system, 178 source split; R1 first-order upwind):
//   eps_{b,i,c} = [ C_b th_c/(W tau_b) + share_b Qdot_c/W + v_b sum_{f: g<0} |g_cf,i| eps_up,f ] / [ 1/tau_b + v_b sum_{f: g>0} g_cf,i ]
//   g_cf,i = A_cf (s_i . n_cf) / V_c                                                             (K_i)
// with eps_up,f the neighbour's value (interior face) or the lagged closure value (boundary face, R9).
//
// B200 design: the upwind graph of every direction is levelled once on the host
// (Kahn, R16: per DIRECTION -- the union graph of an octant is cyclic on the config-4 mesh); cells are stored in level
// order, e is [direction][position][band] so that a cell's bands are one contiguous chunk.  ONE launch runs the
// whole sweep: a CTA owns (direction, group of BG bands) and walks the levels itself with one CTA barrier per
// level -- no dependent-launch chain (~1,500 levels), upwind chunks are re-read from L2 where the same CTA wrote
// them one level earlier.  The per-(direction, position) geometry records are prefetched one pass ahead.
#include <algorithm>
#include <cstdlib>
#include <map>
#include <numeric>

#include "host_util.h"

struct UnsArgs {
  int32_t D, B, BG, NBG, MI, cpp;   // bands per CTA, band groups, max inflow faces per cell, cells per pass
  int32_t rcap;                     // positions held by the shared-memory ring (power of two)
  // staged variant (sweep_unstructured_staged_kernel)
  int32_t st_BG, st_NBG, st_threads, st_vr, st_rr, st_sr;  // bands per CTA, groups, threads, ring capacities (powers of two)
  char *st_rec;                     // [D][e_stride] records of st_rsb bytes: theta, Qdot, outflow sum, inflow
                                    // coefficients [MI], upwind codes [MI] (theta refreshed before every sweep)
  int32_t st_rsb;
  const int32_t *side_ptr;          // [D][l_max+2] first side entry of each level (per direction)
  const int32_t *side_src;          // per direction from side_base[d]: >= 0 position in e, < 0: -1 - inflow index
  const int64_t *side_base;         // [D]
  int32_t n_act, l_max;
  int64_t e_stride;                 // positions per direction (n_act rounded up)
  const int32_t *n_lvl;             // [D]
  const int32_t *lvl_ptr;           // [D][l_max+1] first position of each level
  const int32_t *cell;              // [D][e_stride] active cell at a position
  const int32_t *up;                // [MI][D][e_stride] position of the upwind cell, -1-k = inflow value k, INT_MIN = none
  const double *gin;                // [MI][D][e_stride] |g| of the inflow face
  const double *gout;               // [D][e_stride] sum of g over the outflow faces
  const double *theta, *Qdot;       // [n_act]
  const double *kA, *kS, *itau, *vb;  // [B] C_b/(W tau_b), share_b/W, 1/tau_b, v_b
  const double *bin;
  const int64_t *dir_bin;
  const int32_t *dir_nin;
  double *e;
  // moments
  const int32_t *a2pos;             // [D][n_act]
  const double *w, *s;              // [D], [D][3]
  double *theta_SI, *theta_en, *q;
  double beta, Csum;
};

namespace {

constexpr int32_t kNone = INT32_MIN;

// ---- (a5) the sweep -----------------------------------------------------------------------------------------------------
// Upwind references carry their class in the top bits (decided once at create):
//   kUpRing  the upwind cell lies within the last `rcap` positions before the end of this cell's level: its value is
//            still in the CTA's shared-memory ring (positions are written in increasing order, slot = pos mod rcap);
//   kUpOld   the upwind cell's level is at least 3 levels back: final and visible long before this cell's turn, so
//            the value is fetched from global memory a whole item ahead, off the per-level critical path;
//   neither  (a level wider than the ring) read from global memory after the level barrier.
// Per thread the work items (its cells, in level order) run through a three-stage pipeline: geometry record two
// items ahead, operand values (theta, Qdot, inflow, old upwind values) one item ahead, compute now.  Between two
// level barriers a thread therefore touches only registers and shared memory.
constexpr int32_t kUpRing = 1 << 29, kUpOld = 1 << 28, kUpMask = (1 << 28) - 1;

template <int MI>
__global__ void __launch_bounds__(256, 3) sweep_unstructured_kernel(const UnsArgs a) {
  extern __shared__ double ring[];  // [rcap][BG]
  const int d = blockIdx.x / a.NBG, bg = blockIdx.x % a.NBG;
  const int slot0 = threadIdx.x / a.BG, bl = threadIdx.x - slot0 * a.BG;
  const int b = bg * a.BG + bl;
  const bool live = b < a.B && slot0 < a.cpp;
  const int bb = min(b, a.B - 1);
  const double kA = a.kA[bb], kS = a.kS[bb], itau = a.itau[bb], vb = a.vb[bb];
  const int64_t dbase = (int64_t)d * a.e_stride;
  double *const ed = a.e + dbase * a.B + bb;             // + pos * B
  const double *const bind = a.bin + a.dir_bin[d] + (int64_t)bb * a.dir_nin[d];
  const int32_t *const cell = a.cell + dbase;
  const double *const gout = a.gout + dbase;
  const int32_t *const lp = a.lvl_ptr + (int64_t)d * (a.l_max + 1);
  const int64_t kstride = (int64_t)a.D * a.e_stride;
  const int n_lvl = a.n_lvl[d], cpp = a.cpp;
  const int rmask = a.rcap - 1, BG = a.BG;

  struct Rec {
    int c, pos, lvl;
    double go;
    int up[MI];
    double gi[MI];
  };
  auto fetch_rec = [&](Rec &r, int pos, int lvl) {
    r.pos = pos;
    r.lvl = lvl;
    r.c = __ldg(cell + pos);
    r.go = __ldg(gout + pos);
#pragma unroll
    for (int k = 0; k < MI; ++k) {
      r.up[k] = __ldg(a.up + k * kstride + dbase + pos);
      r.gi[k] = __ldg(a.gin + k * kstride + dbase + pos);
    }
  };
  // item cursor: the thread's next position at or after p in level order (n_lvl = exhausted)
  int cl = 0, clo = lp[0], chi = n_lvl > 0 ? lp[1] : 0, cp = clo + slot0;
  auto settle = [&]() {
    while (cp >= chi && cl < n_lvl) {
      ++cl;
      if (cl < n_lvl) {
        clo = chi;
        chi = lp[cl + 1];
        cp = clo + slot0;
      }
    }
  };
  auto advance = [&]() {
    cp += cpp;
    settle();
  };
  constexpr int QD = 1;   // records in flight behind stage V (deeper queues spill under the 3-CTA register cap)
  Rec rV{}, rQ[QD];       // stage V: record arrived, values (being) fetched; rQ: records in flight, oldest first
  bool hasV = false, vIssued = false;
  int nQ = 0;
  double thV = 0.0, qV = 0.0, valV[MI];
  auto issue_vals = [&]() {  // operands of stage V that do not depend on the sweep's recent output
    thV = a.theta[rV.c];
    qV = a.Qdot[rV.c];
#pragma unroll
    for (int k = 0; k < MI; ++k) {
      const int u = rV.up[k];
      valV[k] = 0.0;
      if (u != kNone) {
        if (u < 0) valV[k] = bind[-1 - u];
        else if (u & kUpOld) valV[k] = ed[(int64_t)(u & kUpMask) * a.B];
      }
    }
    vIssued = true;
  };
  if (live) {
    settle();
    if (cl < n_lvl) { fetch_rec(rV, cp, cl); hasV = true; advance(); }
#pragma unroll
    for (int j = 0; j < QD; ++j)
      if (cl < n_lvl) { fetch_rec(rQ[j], cp, cl); nQ = j + 1; advance(); }
  }

  for (int l = 0; l < n_lvl; ++l) {
    // levels <= l-1 are complete and visible here
    if (hasV && !vIssued && rV.lvl <= l + 2) issue_vals();
    while (hasV && rV.lvl == l) {
      if (!vIssued) issue_vals();
      const int pos = rV.pos;
      double num = kA * thV + kS * qV;
      const double den = itau + vb * rV.go;
#pragma unroll
      for (int k = 0; k < MI; ++k) {
        const int u = rV.up[k];
        if (u != kNone) {
          double val = valV[k];
          if (u >= 0 && !(u & kUpOld)) {
            const int up = u & kUpMask;
            val = (u & kUpRing) ? ring[(up & rmask) * BG + bl] : ed[(int64_t)up * a.B];
          }
          num += vb * rV.gi[k] * val;
        }
      }
      const double res = num / den;
      ed[(int64_t)pos * a.B] = res;
      ring[(pos & rmask) * BG + bl] = res;
      // shift the pipeline
      hasV = nQ > 0;
      vIssued = false;
      if (hasV) {
        rV = rQ[0];
#pragma unroll
        for (int j = 0; j + 1 < QD; ++j) rQ[j] = rQ[j + 1];
        --nQ;
        if (cl < n_lvl) {  // the queue is full whenever items remain, so the new record goes to the last slot
          fetch_rec(rQ[QD - 1], cp, cl);
          ++nQ;
          advance();
        }
        if (rV.lvl <= l + 2) issue_vals();
      }
    }
    __syncthreads();  // level l is visible to the whole CTA (it alone reads these rows)
  }
}

// ---- (a5) staged variant --------------------------------------------------------------------------------------------
// Same arithmetic, but between two level barriers a thread touches only shared memory:
//   * the per-position records (theta and Qdot pre-permuted per direction, outflow sum, inflow coefficients, upwind
//     codes) stream into a ring of `rr` positions by cp.async, up to rr positions ahead of the level in progress;
//   * an upwind value is read from the value ring (the last `vr` outputs), or -- wall inflow and upwind cells at
//     least 3 levels back -- from a side ring that cp.async fills 2 levels ahead (the sources are final by then);
//     the rare reference in between (a level wider than the ring) is a global load after the barrier.
//   * one CTA per SM: (direction, group of bands) with 32 cells per pass; every thread issues its share of the
//     copies at the top of a level, commits one group per level and waits for the previous level's group before
//     the barrier, so a copy has a level time to land.  create() checks the spans that make this safe
//     (3 consecutive levels fit the record ring, their side entries the side ring) and falls back otherwise.
// upwind codes: >= 0 shared-memory offset (slot * BG) in the value ring or the side ring behind it; kStLate (sign bit
// set, != kNone): position in e, or with kStIn an index into the band's inflow row
constexpr int32_t kStLate = INT32_MIN | (1 << 30), kStIn = 1 << 27, kStMask = (1 << 27) - 1;

__device__ __forceinline__ void cp_async8(void *dst, const void *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

__global__ void theta_permute_kernel(const UnsArgs a) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)a.D * a.e_stride) return;
  const int pos = (int)(i % a.e_stride);
  if (pos < a.n_act) *reinterpret_cast<double *>(a.st_rec + i * a.st_rsb) = a.theta[a.cell[i]];
}

template <int MI>
__global__ void __launch_bounds__(640, 1) sweep_unstructured_staged_kernel(const UnsArgs a) {
  extern __shared__ __align__(16) unsigned char st_smem[];
  const int BG = a.st_BG, VR = a.st_vr, RR = a.st_rr, SR = a.st_sr;
  double *vring = reinterpret_cast<double *>(st_smem);  // [VR][BG]
  double *side = vring + (size_t)VR * BG;                // [SR][BG]
  constexpr int RSB = (24 + 12 * MI + 15) / 16 * 16, NQ = RSB / 16;  // record: th, q, go, gi[MI] doubles, up[MI] ints
  char *rec_s = reinterpret_cast<char *>(side + (size_t)SR * BG);  // [RR] records
  const int d = blockIdx.x / a.st_NBG, bg = blockIdx.x % a.st_NBG;
  const int tid = threadIdx.x, nth = blockDim.x;
  const int slot0 = tid / BG, bl = tid - slot0 * BG;
  const int b = bg * BG + bl;
  const bool live = b < a.B && slot0 < 32;
  const int bb = min(b, a.B - 1);
  const double kA = a.kA[bb], kS = a.kS[bb], itau = a.itau[bb], vb = a.vb[bb];
  const int64_t dbase = (int64_t)d * a.e_stride;
  double *const ed = a.e + dbase * a.B + bb;
  const int64_t nin = a.dir_nin[d];
  const double *const bin_b = a.bin + a.dir_bin[d] + (int64_t)bb * nin;
  const int32_t *const lp = a.lvl_ptr + (int64_t)d * (a.l_max + 1);
  const int32_t *const sp = a.side_ptr + (int64_t)d * (a.l_max + 2);
  const int32_t *const ssrc = a.side_src + a.side_base[d];
  const int n_lvl = a.n_lvl[d], n_act = a.n_act;

  int pf = 0, sf = 0;  // next record position / side entry to request (identical in every thread)
  // Side copies: the thread (cell slot slot0, band bl) copies band bl of the entries sf + slot0, sf + slot0 + 32, ...
  // (no index arithmetic beyond an add); the sources of the next level's first two are prefetched into registers.
  constexpr int PRE = 2;
  int pre_src[PRE], pre_sf = -1;
  auto prefetch_src = [&](int s0, int s1) {
    pre_sf = s0;
#pragma unroll
    for (int i = 0; i < PRE; ++i) {
      const int e = s0 + slot0 + 32 * i;
      pre_src[i] = (live && e < s1) ? __ldg(ssrc + e) : 0;
    }
  };
  auto issue = [&](int pf_end, int sf_end) {
    for (int p = pf + tid; p < pf_end; p += nth) {
      const int s = p & (RR - 1);
      const char *src = a.st_rec + (dbase + p) * RSB;
#pragma unroll
      for (int i = 0; i < NQ; ++i) cp_async16(rec_s + (size_t)s * RSB + 16 * i, src + 16 * i);
    }
    pf = max(pf, pf_end);
    if (live) {
      const bool hit = pre_sf == sf;
      int i = 0;
      for (int e = sf + slot0; e < sf_end; e += 32, ++i) {
        const int src = (hit && i < PRE) ? (i == 0 ? pre_src[0] : pre_src[1]) : __ldg(ssrc + e);
        const double *from = src >= 0 ? ed + (int64_t)src * a.B : bin_b + (-1 - src);
        cp_async8(side + (size_t)(e & (SR - 1)) * BG + bl, from);
      }
    }
    sf = max(sf, sf_end);
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // prologue: everything the first levels need, fully landed
  issue(min(n_act, RR), min(sp[min(2, n_lvl)], SR));
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  // level table entries one level ahead in registers: no global load sits between a barrier and the level's work
  int lo = lp[0], hi = n_lvl > 0 ? lp[1] : 0, hi_n = lp[min(2, n_lvl)];
  int sp_l = sp[0], sp_l4 = sp[min(3, n_lvl)], sp_n = sp[min(1, n_lvl)], sp_n4 = sp[min(4, n_lvl)];
  prefetch_src(sf, max(sf, min(sp_l4, sp_l + SR)));
  __syncthreads();

  for (int l = 0; l < n_lvl; ++l) {
    issue(min(n_act, lo + RR), min(sp_l4, sp_l + SR));
    // next level's table entries and side sources, in flight while this level is computed
    const int hi_nn = lp[min(l + 3, n_lvl)];
    const int sp_nn = sp[min(l + 2, n_lvl)], sp_nn4 = sp[min(l + 5, n_lvl)];
    prefetch_src(sf, max(sf, min(sp_n4, sp_n + SR)));
    if (live) {
      double *ep = ed + (int64_t)(lo + slot0) * a.B;  // this thread's output, advanced by pointer (no 64-bit multiply per cell)
      for (int pos = lo + slot0; pos < hi; pos += 32, ep += 32 * (int64_t)a.B) {
        const int s = pos & (RR - 1);
        // the whole record in NQ 16-byte shared-memory loads
        uint4 raw[NQ];
#pragma unroll
        for (int i = 0; i < NQ; ++i) raw[i] = reinterpret_cast<const uint4 *>(rec_s + (size_t)s * RSB)[i];
        double rd[3 + MI];
        int32_t ru[MI];
        memcpy(rd, raw, sizeof(rd));
        memcpy(ru, reinterpret_cast<const char *>(raw) + sizeof(rd), sizeof(ru));
        double num = kA * rd[0] + kS * rd[1];
        const double den = itau + vb * rd[2];
#pragma unroll
        for (int k = 0; k < MI; ++k) {
          const int u = ru[k];
          if (u != kNone) {
            // ring and side references carry their shared-memory offset (slot * BG) ready-made; the rest is late
            const double val = u >= 0 ? vring[u + bl] : (u & kStIn) ? bin_b[u & kStMask] : ed[(int64_t)(u & kStMask) * a.B];
            num += vb * rd[3 + k] * val;
          }
        }
        const double res = num * __drcp_rn(den);  // within 1 ulp of num / den
        *ep = res;
        vring[(size_t)(pos & (VR - 1)) * BG + bl] = res;
      }
    }
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    __syncthreads();
    lo = hi; hi = hi_n; hi_n = hi_nn;
    sp_l = sp_n; sp_l4 = sp_n4; sp_n = sp_nn; sp_n4 = sp_nn4;
  }
}

// ---- (a6) moments in the per-direction layout: one warp per cell; a lane is (direction within a group of 4, band
// modulo 8), so every 8-lane group reads 64 contiguous bytes of one (direction, cell) chunk and all lanes stay busy for
// any band count; the direction loop is unrolled for memory-level parallelism.  Fixed shuffle tree: deterministic.
__global__ void __launch_bounds__(256) moments_unstructured_kernel(const UnsArgs a) {
  extern __shared__ double sm[];  // w[D], w s[D][3], 1/tau[B], v[B]
  double *wsm = sm, *wss = sm + a.D, *its = sm + 4 * a.D, *vbs = its + a.B;
  for (int k = threadIdx.x; k < a.D; k += blockDim.x) wsm[k] = a.w[k];
  for (int k = threadIdx.x; k < 3 * a.D; k += blockDim.x) wss[k] = a.w[k / 3] * a.s[k];
  for (int k = threadIdx.x; k < a.B; k += blockDim.x) { its[k] = a.itau[k]; vbs[k] = a.vb[k]; }
  __syncthreads();
  const int lane = threadIdx.x & 31, dl = lane >> 3, b8 = lane & 7;
  const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (c >= a.n_act) return;
  double A1 = 0.0, A2 = 0.0, qx = 0.0, qy = 0.0, qz = 0.0;
  for (int d0 = 0; d0 < a.D; d0 += 16) {  // 4 direction groups of 4 in flight
    int64_t base[4];
    int dd[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      dd[u] = d0 + 4 * u + dl;
      base[u] = dd[u] < a.D ? ((int64_t)dd[u] * a.e_stride + __ldg(a.a2pos + (int64_t)dd[u] * a.n_act + c)) * a.B : -1;
    }
    constexpr int KB = 3;  // band chunks of 8 in flight on top of the 4 direction groups: 12 loads per lane before the first use (5: slower)
    for (int b0 = 0; b0 < a.B; b0 += 8 * KB) {
      double v[KB][4];
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        const int b = b0 + 8 * k + b8;
#pragma unroll
        for (int u = 0; u < 4; ++u) v[k][u] = (b < a.B && base[u] >= 0) ? __ldcs(a.e + base[u] + b) : 0.0;
      }
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        const int b = b0 + 8 * k + b8;
        if (b < a.B) {
          const double it = its[b], vb = vbs[b];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (base[u] >= 0) {
              const double wv = wsm[dd[u]] * v[k][u];
              A1 += it * wv;                            // Eq. 5 numerator
              A2 += wv;                                 // R13
              qx += vb * (wss[3 * dd[u]] * v[k][u]);    // Eq. 7
              qy += vb * (wss[3 * dd[u] + 1] * v[k][u]);
              qz += vb * (wss[3 * dd[u] + 2] * v[k][u]);
            }
          }
        }
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    A1 += __shfl_xor_sync(0xffffffffu, A1, o);
    A2 += __shfl_xor_sync(0xffffffffu, A2, o);
    qx += __shfl_xor_sync(0xffffffffu, qx, o);
    qy += __shfl_xor_sync(0xffffffffu, qy, o);
    qz += __shfl_xor_sync(0xffffffffu, qz, o);
  }
  if (lane == 0) {
    a.theta_SI[c] = A1 / a.beta;
    a.theta_en[c] = A2 / a.Csum;
    a.q[3 * (int64_t)c] = qx;
    a.q[3 * (int64_t)c + 1] = qy;
    a.q[3 * (int64_t)c + 2] = qz;
  }
}

// ---- (a8) theta <- theta_SI (mode 0) or theta_SI + delta (mode 1), max |dT| -----------------------------------------------------
__global__ void __launch_bounds__(256) update_unstructured_kernel(int n, int mode, const double *theta_SI, const double *x,
                                                                  double *theta, double *theta_prev, unsigned long long *maxdT) {
  __shared__ double red[8];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  double dlt = 0.0;
  if (i < n) {
    if (mode == 0) theta_prev[i] = theta[i];
    const double th = mode == 0 ? theta_SI[i] : theta_SI[i] + x[i];
    theta[i] = th;
    dlt = fabs(th - theta_prev[i]);
  }
  auto nanmax = [](double p, double q) { return !(q <= p) ? q : p; };
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dlt = nanmax(dlt, __shfl_xor_sync(0xffffffffu, dlt, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = dlt;
  __syncthreads();
  if (threadIdx.x < 32) {
    dlt = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dlt = nanmax(dlt, __shfl_xor_sync(0xffffffffu, dlt, o));
    if (threadIdx.x == 0) atomicMax(maxdT, (unsigned long long)__double_as_longlong(dlt));
  }
}

typedef void (*uns_fn)(const UnsArgs);
uns_fn pick_uns(int mi) {
  switch (mi) {
    case 1: return sweep_unstructured_kernel<1>;
    case 2: return sweep_unstructured_kernel<2>;
    case 3: return sweep_unstructured_kernel<3>;
    case 4: return sweep_unstructured_kernel<4>;
    case 5: return sweep_unstructured_kernel<5>;
    case 6: return sweep_unstructured_kernel<6>;
    case 7: return sweep_unstructured_kernel<7>;
  }
  return nullptr;
}

}  // namespace

typedef void (*uns_st_fn)(const UnsArgs);
static uns_st_fn pick_uns_staged(int mi) {
  switch (mi) {
    case 1: return sweep_unstructured_staged_kernel<1>;
    case 2: return sweep_unstructured_staged_kernel<2>;
    case 3: return sweep_unstructured_staged_kernel<3>;
    case 4: return sweep_unstructured_staged_kernel<4>;
  }
  return nullptr;
}

int nb_launch_sweep_unstructured(nanobte_solver *h) {
  const UnsArgs &a = *h->uns;
  if (h->uns_staged) {
    uns_st_fn fs = pick_uns_staged(a.MI);
    const int64_t n = (int64_t)a.D * a.e_stride;
    theta_permute_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(a);
    h->launches++;
    // per-function attribute, shared by every solver in the process: set before every launch
    NB_CUDA(h, cudaFuncSetAttribute(fs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->sweep_smem));
    fs<<<a.D * a.st_NBG, a.st_threads, h->sweep_smem, h->stream>>>(a);
    h->launches++;
    NB_CUDA(h, cudaGetLastError());
    return 0;
  }
  uns_fn fn = pick_uns(a.MI);
  if (!fn) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "cells with more than 7 inflow faces are not supported");
  NB_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(h->sweep_smem, 1024)));
  fn<<<a.D * a.NBG, h->sweep_threads, h->sweep_smem, h->stream>>>(a);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

int nb_launch_moments_unstructured(nanobte_solver *h) {
  const UnsArgs &a = *h->uns;
  const int wpb = 8;
  moments_unstructured_kernel<<<(a.n_act + wpb - 1) / wpb, wpb * 32, ((size_t)4 * a.D + 2 * a.B) * sizeof(double), h->stream>>>(a);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

int nb_launch_update_unstructured(nanobte_solver *h, int mode) {
  update_unstructured_kernel<<<(h->n_act + 255) / 256, 256, 0, h->stream>>>(h->n_act, mode, h->theta_SI, h->cg_x, h->theta,
                                                                           h->theta_prev, h->d_maxdT);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  return 0;
}

void nb_free_unstructured(nanobte_solver *h) {
  delete h->uns;
  h->uns = nullptr;
}

// =====================================================================================================================
// (a1) host setup
// =====================================================================================================================
namespace {

int build_uns(nanobte_solver *h, const nanobte_unstructured_mesh *m, const nanobte_bands *bands, const nanobte_quadrature *quad,
              const nanobte_tag *tags, int n_tags, const double *Qdot, const nanobte_options *opt, bool size_only,
              size_t *bytes_out) {
  if (!m || !opt) return nb_fail(h, NANOBTE_E_INVALID, "null argument");
  const int nn = m->n_nodes, nc = m->n_cells;
  if (nn < 3 || nc < 1 || !m->xy || !m->cell_ptr || !m->cell_nodes) return nb_fail(h, NANOBTE_E_INVALID, "bad mesh");
  Common cm;
  int rc = nb_validate_common(h, 2, bands, quad, tags, n_tags, cm);
  if (rc) return rc;
  // band shard: the sums over the whole band table come from the caller (nanobte_options)
  if (opt->beta_total > 0.0) cm.beta = opt->beta_total;
  if (opt->Csum_total > 0.0) {
    cm.Csum = opt->Csum_total;
    if (bands->src_share == nullptr)  // source shares of the shard's bands in the whole table (R5)
      for (int b = 0; b < cm.B; ++b) cm.share[b] = cm.C[b] / cm.Csum;
  }
  if (opt->kappa_total > 0.0) cm.kappa = opt->kappa_total;
  const int B = cm.B, D = cm.D;
  const int nf = m->cell_ptr[nc];
  if (m->cell_ptr[0] != 0 || nf < 3 * nc) return nb_fail(h, NANOBTE_E_INVALID, "bad cell_ptr");

  // ---- geometry: area, centroid, edge length / outward normal / centroid distance; edge matching ---------------------------
  std::vector<double> vol(nc), cen(2 * (size_t)nc), flen(nf), fnx(nf), fny(nf), fdist(nf);
  std::vector<int32_t> fnbr(nf, -1), fbf(nf, -1), fcell(nf);
  std::map<std::pair<int, int>, int> open_edge;  // (lo, hi) -> face waiting for its partner
  std::vector<char> matched(nf, 0);
  for (int c = 0; c < nc; ++c) {
    const int p0 = m->cell_ptr[c], np = m->cell_ptr[c + 1] - p0;
    if (np < 3) return nb_fail(h, NANOBTE_E_INVALID, "cell %d has fewer than 3 nodes", c);
    double a2 = 0, sx = 0, sy = 0;
    for (int k = 0; k < np; ++k) {
      const int n0 = m->cell_nodes[p0 + k], n1 = m->cell_nodes[p0 + (k + 1) % np];
      if (n0 < 0 || n0 >= nn || n1 < 0 || n1 >= nn) return nb_fail(h, NANOBTE_E_INVALID, "cell %d: bad node id", c);
      const double x0 = m->xy[2 * n0], y0 = m->xy[2 * n0 + 1], x1 = m->xy[2 * n1], y1 = m->xy[2 * n1 + 1];
      const double cr = x0 * y1 - x1 * y0;
      a2 += cr;
      sx += (x0 + x1) * cr;
      sy += (y0 + y1) * cr;
    }
    if (!(a2 > 0)) return nb_fail(h, NANOBTE_E_INVALID, "cell %d is not counter-clockwise (area %g)", c, 0.5 * a2);
    vol[c] = 0.5 * a2;  // unit depth
    cen[2 * c] = sx / (3.0 * a2);
    cen[2 * c + 1] = sy / (3.0 * a2);
    for (int k = 0; k < np; ++k) {
      const int f = p0 + k, n0 = m->cell_nodes[p0 + k], n1 = m->cell_nodes[p0 + (k + 1) % np];
      const double ex = m->xy[2 * n1] - m->xy[2 * n0], ey = m->xy[2 * n1 + 1] - m->xy[2 * n0 + 1];
      const double len = std::sqrt(ex * ex + ey * ey);
      if (!(len > 0)) return nb_fail(h, NANOBTE_E_INVALID, "cell %d has a zero-length edge", c);
      flen[f] = len;
      fnx[f] = ey / len;  // outward normal of a counter-clockwise polygon edge
      fny[f] = -ex / len;
      fcell[f] = c;
      fdist[f] = (m->xy[2 * n0] - cen[2 * c]) * fnx[f] + (m->xy[2 * n0 + 1] - cen[2 * c + 1]) * fny[f];
      const std::pair<int, int> key(std::min(n0, n1), std::max(n0, n1));
      auto it = open_edge.find(key);
      if (it == open_edge.end()) {
        open_edge.emplace(key, f);
      } else {
        const int g = it->second;
        if (matched[g]) return nb_fail(h, NANOBTE_E_INVALID, "edge (%d,%d) is shared by more than two cells", key.first, key.second);
        matched[g] = matched[f] = 1;
        fnbr[f] = fcell[g];
        fnbr[g] = c;
      }
    }
  }
  for (int f = 0; f < nf; ++f)
    if (fnbr[f] >= 0) {
      const int c0 = fcell[f], c1 = fnbr[f];
      const double dx = cen[2 * c1] - cen[2 * c0], dy = cen[2 * c1 + 1] - cen[2 * c0 + 1];
      fdist[f] = std::sqrt(dx * dx + dy * dy);
    }

  // ---- boundary faces ------------------------------------------------------------------------------------------------------
  const int nbf = m->n_bfaces;
  if (nbf < 0 || (nbf > 0 && (!m->bf_nodes || !m->bf_tag))) return nb_fail(h, NANOBTE_E_INVALID, "bad boundary face arrays");
  GenericTables G;
  G.act2cell.resize(nc);
  std::iota(G.act2cell.begin(), G.act2cell.end(), 0);
  G.cell2act = G.act2cell;
  G.bf_act.resize(nbf); G.bf_type.resize(nbf); G.bf_p.resize(nbf); G.bf_den.resize(nbf); G.bf_area.resize(nbf); G.bf_eps_w.resize(nbf);
  std::vector<int32_t> bf_face(nbf);
  h->h_bf_tag.assign(m->bf_tag, m->bf_tag + nbf);
  for (int bf = 0; bf < nbf; ++bf) {
    const int n0 = m->bf_nodes[2 * bf], n1 = m->bf_nodes[2 * bf + 1];
    auto it = open_edge.find(std::make_pair(std::min(n0, n1), std::max(n0, n1)));
    if (it == open_edge.end()) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: no such edge", bf);
    const int f = it->second;
    if (matched[f]) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d is an interior edge", bf);
    if (fbf[f] >= 0) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d listed twice", bf);
    const int tg = m->bf_tag[bf];
    if (tg < 0 || tg >= n_tags) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: bad tag", bf);
    const double p = m->bf_p ? m->bf_p[bf] : 0.0;
    if (p < 0 || p > 1) return nb_fail(h, NANOBTE_E_INVALID, "boundary face %d: specularity outside [0,1]", bf);
    fbf[f] = bf;
    bf_face[bf] = f;
    G.bf_act[bf] = fcell[f];
    G.bf_type[bf] = cm.tag_type[tg];
    G.bf_p[bf] = p;
    G.bf_eps_w[bf] = cm.tag_T[tg] - opt->T_ref;
    G.bf_area[bf] = flen[f];
  }
  for (int f = 0; f < nf; ++f)
    if (fnbr[f] < 0 && fbf[f] < 0)
      return nb_fail(h, NANOBTE_E_UNTAGGED, "cell %d has an exposed face without a boundary tag", fcell[f]);

  // ---- per direction: levels (Kahn), positions, sweep records, inflow lists ----------------------------------------------------
  const int64_t e_stride = ((int64_t)nc + 31) / 32 * 32;
  std::vector<int32_t> a2pos((size_t)D * nc), n_lvl(D), cellat((size_t)D * e_stride, 0);
  std::vector<std::vector<int32_t>> lvl_ptrs(D);
  std::vector<double> gout((size_t)D * e_stride, 0.0);
  G.bf_sn.assign((size_t)nbf * D, 0.0);
  G.bf_mirror.assign((size_t)nbf * D, -1);
  G.bf_inidx.assign((size_t)nbf * D, -1);
  G.bf_opos.assign((size_t)nbf * D, -1);
  G.dir_bin.resize(D); G.dir_nin.resize(D); G.dir_row0.resize(D);
  int MI = 1, l_max = 0;
  // pass 1: levels and positions
  std::vector<int32_t> level(nc), indeg(nc), queue(nc);
  std::vector<std::vector<double>> sn_all;  // s_d . n_f for every face, per direction, kept only transiently
  for (int d = 0; d < D; ++d) {
    const double sx = cm.s[3 * d], sy = cm.s[3 * d + 1];
    for (int c = 0; c < nc; ++c) {
      int in = 0, nin_faces = 0;
      for (int f = m->cell_ptr[c]; f < m->cell_ptr[c + 1]; ++f) {
        const double sn = sx * fnx[f] + sy * fny[f];
        if (sn < 0) {
          ++nin_faces;
          if (fnbr[f] >= 0) ++in;
        }
      }
      indeg[c] = in;
      MI = std::max(MI, nin_faces);
    }
    int head = 0, tail = 0;
    for (int c = 0; c < nc; ++c)
      if (indeg[c] == 0) { level[c] = 0; queue[tail++] = c; }
    int lmax_d = 0;
    while (head < tail) {
      const int c = queue[head++];
      lmax_d = std::max(lmax_d, level[c]);
      for (int f = m->cell_ptr[c]; f < m->cell_ptr[c + 1]; ++f) {
        const int nb = fnbr[f];
        if (nb >= 0 && sx * fnx[f] + sy * fny[f] > 0) {  // c is upwind of nb; nb's level is fixed by its LAST upwind cell
          if (--indeg[nb] == 0) { level[nb] = level[c] + 1; queue[tail++] = nb; }
        }
      }
    }
    if (tail != nc) return nb_fail(h, NANOBTE_E_CYCLE, "upwind graph of direction %d is cyclic (%d of %d cells ordered)", d, tail, nc);
    // Kahn's queue pops cells in non-decreasing level order, so level[c] above is the longest upwind path.
    n_lvl[d] = lmax_d + 1;
    l_max = std::max(l_max, n_lvl[d]);
    std::vector<int32_t> &lp = lvl_ptrs[d];
    lp.assign(n_lvl[d] + 1, 0);
    for (int c = 0; c < nc; ++c) lp[level[c] + 1]++;
    for (int l = 0; l < n_lvl[d]; ++l) lp[l + 1] += lp[l];
    std::vector<int32_t> fill(lp.begin(), lp.end() - 1);
    for (int c = 0; c < nc; ++c) {  // cells of a level in cell-id order
      const int pos = fill[level[c]]++;
      a2pos[(size_t)d * nc + c] = pos;
      cellat[(size_t)d * e_stride + pos] = c;
    }
  }
  if (MI > 7) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "a cell has %d inflow faces; at most 7 are supported", MI);
  // pass 2: records
  std::vector<int32_t> up((size_t)MI * D * e_stride, kNone);
  std::vector<double> gin((size_t)MI * D * e_stride, 0.0);
  int64_t bin_total = 0;
  for (int d = 0; d < D; ++d) {
    const double sx = cm.s[3 * d], sy = cm.s[3 * d + 1];
    int nin = 0;
    G.dir_bin[d] = bin_total;
    G.dir_row0[d] = d * B;
    for (int c = 0; c < nc; ++c) {
      const int64_t at = (int64_t)d * e_stride + a2pos[(size_t)d * nc + c];
      int k = 0;
      double go = 0.0;
      for (int f = m->cell_ptr[c]; f < m->cell_ptr[c + 1]; ++f) {
        const double sn = sx * fnx[f] + sy * fny[f];
        const double g = flen[f] * sn / vol[c];  // O1
        if (g > 0) {
          go += g;
        } else if (g < 0) {
          const int64_t r = (int64_t)k * D * e_stride + at;
          gin[r] = -g;
          if (fnbr[f] >= 0) {
            up[r] = a2pos[(size_t)d * nc + fnbr[f]];
          } else {
            up[r] = -1 - nin;
            G.bf_inidx[(size_t)fbf[f] * D + d] = nin++;
          }
          ++k;
        }
      }
      gout[at] = go;
    }
    G.dir_nin[d] = nin;
    bin_total += (int64_t)B * nin;
  }
  G.bin_total = bin_total;

  // ---- closure tables -------------------------------------------------------------------------------------------------------
  for (int bf = 0; bf < nbf; ++bf) {
    const int f = bf_face[bf];
    const double nrm[3] = {fnx[f], fny[f], 0.0};
    const bool refl = G.bf_type[bf] == NANOBTE_SPECULAR || G.bf_type[bf] == NANOBTE_MIXED;
    double den = 0.0;
    for (int d = 0; d < D; ++d) {
      const double sn = cm.s[3 * d] * nrm[0] + cm.s[3 * d + 1] * nrm[1] + cm.s[3 * d + 2] * nrm[2];
      G.bf_sn[(size_t)bf * D + d] = sn;
      if (sn < 0) {
        den += cm.w[d] * (-sn);
        if (refl) {
          const int mj = nb_find_mirror(cm, d, nrm);
          if (mj < 0) return nb_fail(h, NANOBTE_E_SPECULAR, "boundary face %d: mirror image of direction %d is not in the quadrature", bf, d);
          G.bf_mirror[(size_t)bf * D + d] = mj;
        }
      } else if (sn > 0) {
        G.bf_opos[(size_t)bf * D + d] = a2pos[(size_t)d * nc + fcell[f]];
      }
    }
    G.bf_den[bf] = den;
  }

  // ---- cells: volumes, source, initial theta, diffusion stencil (two-point flux, R14e) ------------------------------------------
  int maxf = 0;
  for (int c = 0; c < nc; ++c) maxf = std::max(maxf, m->cell_ptr[c + 1] - m->cell_ptr[c]);
  G.vol = vol;
  G.Qdot_act.resize(nc); G.theta0.resize(nc);
  G.cg_nf = maxf;
  G.cg_nbr.assign((size_t)maxf * nc, 0);
  G.cg_coef.assign((size_t)maxf * nc, 0.0);
  G.cg_diag.assign(nc, 0.0);
  G.fourier_rhs.assign(nc, 0.0);
  G.cellbf_ptr.assign(nc + 1, 0);
  G.cg_xyz.assign((size_t)3 * nc, 0.0);
  for (int c = 0; c < nc; ++c) {
    G.cg_xyz[3 * (size_t)c] = cen[2 * c];
    G.cg_xyz[3 * (size_t)c + 1] = cen[2 * c + 1];
    G.Qdot_act[c] = Qdot ? Qdot[c] : 0.0;
    G.fourier_rhs[c] = G.vol[c] * G.Qdot_act[c];
    G.theta0[c] = opt->T_init ? opt->T_init[c] - opt->T_ref : 0.0;
    for (int k = 0; k < maxf; ++k) G.cg_nbr[(size_t)k * nc + c] = c;
    int k = 0;
    for (int f = m->cell_ptr[c]; f < m->cell_ptr[c + 1]; ++f, ++k) {
      if (fnbr[f] >= 0) {
        const double cf = cm.kappa * flen[f] / fdist[f];
        G.cg_nbr[(size_t)k * nc + c] = fnbr[f];
        G.cg_coef[(size_t)k * nc + c] = cf;
        G.cg_diag[c] += cf;
      } else if (G.bf_type[fbf[f]] == NANOBTE_THERMALIZING) {
        G.cg_diag[c] += cm.kappa * flen[f] / fdist[f];  // delta = 0 on the wall
        G.fourier_rhs[c] += cm.kappa * flen[f] / fdist[f] * G.bf_eps_w[fbf[f]];  // theta = T_w - T_ref on the wall (R21)
      } else {
        G.cellbf.push_back(fbf[f]);
      }
    }
    G.cellbf_ptr[c + 1] = (int32_t)G.cellbf.size();
  }
  G.tagface_ptr.assign(n_tags + 1, 0);
  for (int bf = 0; bf < nbf; ++bf) G.tagface_ptr[m->bf_tag[bf] + 1]++;
  for (int t = 0; t < n_tags; ++t) G.tagface_ptr[t + 1] += G.tagface_ptr[t];
  G.tagface.resize(nbf);
  {
    std::vector<int> fill(G.tagface_ptr.begin(), G.tagface_ptr.end() - 1);
    for (int bf = 0; bf < nbf; ++bf) G.tagface[fill[m->bf_tag[bf]]++] = bf;
  }

  // ---- launch shape: bands per CTA so that D * NBG CTAs fill the SMs a few times over ------------------------------------------
  int BG = opt->sweep_G > 0 ? std::min(opt->sweep_G, B) : std::min(B, 8);
  if (opt->sweep_G <= 0 && B % 8 != 0 && B <= 12) BG = B;
  const int NBG = (B + BG - 1) / BG;
  int threads = opt->sweep_threads > 0 ? std::min(256, (opt->sweep_threads + 31) / 32 * 32) : 256;
  threads = std::max(threads, (BG + 31) / 32 * 32);
  const int cpp = threads / BG;
  // shared-memory ring of the CTA's most recent outputs: the largest power of two of positions within 64 KB
  int rcap = 64;
  while ((size_t)rcap * 2 * BG * sizeof(double) <= 64 * 1024 && rcap * 2 <= (1 << 20)) rcap *= 2;
  if (nc >= (1 << 28)) return nb_fail(h, NANOBTE_E_UNSUPPORTED, "more than 2^28 cells");
  // class of every upwind reference (see the kernel): ring / old / neither
  {
    std::vector<int32_t> lvl_of(nc);
    for (int d = 0; d < D; ++d) {
      const std::vector<int32_t> &lp = lvl_ptrs[d];
      for (int l = 0; l < n_lvl[d]; ++l)
        for (int pos = lp[l]; pos < lp[l + 1]; ++pos) lvl_of[pos] = l;
      for (int k = 0; k < MI; ++k)
        for (int pos = 0; pos < nc; ++pos) {
          int32_t &u = up[(size_t)k * D * e_stride + (size_t)d * e_stride + pos];
          if (u < 0) continue;  // none or boundary inflow
          const int l = lvl_of[pos];
          if (u >= lp[l + 1] - rcap) u |= kUpRing;
          else if (lvl_of[u] <= l - 3) u |= kUpOld;
        }
    }
  }

  // ---- staged variant: launch shape, upwind codes, side lists, spans ---------------------------------------------------------
  int st_NBG = std::max(1, std::min(B, h->n_sm / std::max(1, D)));
  int st_BG = opt->sweep_G > 0 ? std::min(opt->sweep_G, B) : (B + st_NBG - 1) / st_NBG;
  st_BG = std::min(st_BG, 20);
  st_NBG = (B + st_BG - 1) / st_BG;
  const int st_threads = (32 * st_BG + 31) / 32 * 32;
  // shared-memory budget of the one CTA per SM: record ring (fixed), a side ring of 64 entries, the rest for the value ring
  const size_t st_budget = 225 * 1024;
  const size_t st_rec_smem = (size_t)1024 * ((24 + 12 * MI + 15) / 16 * 16);
  int st_sr = 64, st_vr = 64;
  while (st_rec_smem + (size_t)st_sr * st_BG * sizeof(double) + (size_t)st_vr * 2 * st_BG * sizeof(double) + 64 <= st_budget && st_vr < 4096) st_vr *= 2;
  while (st_rec_smem + (size_t)st_sr * 2 * st_BG * sizeof(double) + (size_t)st_vr * st_BG * sizeof(double) + 64 <= st_budget && st_sr < 1024) st_sr *= 2;
  const int st_rr = 1024;
  bool staged = MI <= 4 && std::getenv("NANOBTE_UNS_PLAIN") == nullptr;
  std::vector<int32_t> st_up(up.size(), kNone), side_ptr((size_t)D * (l_max + 2), 0), side_src;
  std::vector<int64_t> side_base(D, 0);
  long n_late = 0;
  {
    std::vector<int32_t> lvl_of(nc);
    for (int d = 0; d < D && staged; ++d) {
      const std::vector<int32_t> &lp = lvl_ptrs[d];
      for (int l = 0; l < n_lvl[d]; ++l)
        for (int pos = lp[l]; pos < lp[l + 1]; ++pos) lvl_of[pos] = l;
      side_base[d] = (int64_t)side_src.size();
      int32_t ns = 0;
      for (int l = 0; l < n_lvl[d]; ++l) {
        side_ptr[(size_t)d * (l_max + 2) + l] = ns;
        for (int pos = lp[l]; pos < lp[l + 1]; ++pos)
          for (int k = 0; k < MI; ++k) {
            const size_t r = (size_t)k * D * e_stride + (size_t)d * e_stride + pos;
            const int32_t u = up[r] == kNone ? kNone : (up[r] < 0 ? up[r] : (up[r] & kUpMask));
            if (u == kNone) continue;
            if (u >= 0 && u >= lp[l + 1] - st_vr) { st_up[r] = (u & (st_vr - 1)) * st_BG; continue; }  // offset in the value ring
            // wall inflow, or final long before its turn: side ring -- if the entry can be requested in time (entries of
            // level l are requested at level l-2, at most st_sr beyond the first entry of that level)
            const int32_t first = side_ptr[(size_t)d * (l_max + 2) + std::max(0, l - 2)];
            if ((u < 0 || lvl_of[u] <= l - 3) && ns - first < st_sr) {
              st_up[r] = (st_vr + (ns & (st_sr - 1))) * st_BG;  // offset in the side ring, which follows the value ring
              ++ns;
              side_src.push_back(u);
              continue;
            }
            st_up[r] = kStLate | (u < 0 ? (kStIn | (-1 - u)) : u);  // late: global load after the level barrier
            ++n_late;
          }
      }
      for (int l = n_lvl[d]; l < l_max + 2; ++l) side_ptr[(size_t)d * (l_max + 2) + l] = ns;
      if (ns >= (1 << 27) || nc >= (1 << 27)) staged = false;
      for (int l = 0; l < n_lvl[d] && staged; ++l) {  // three consecutive levels must fit the rings
        const int l4 = std::min(l + 3, n_lvl[d]);
        if (lp[l4] - lp[l] > st_rr) staged = false;
      }
    }
  }
  const size_t st_smem = ((size_t)st_vr * st_BG + (size_t)st_sr * st_BG) * sizeof(double) + st_rec_smem + 64;
  if (st_smem > 227 * 1024 - 512) staged = false;
  const int st_rsb = (24 + 12 * MI + 15) / 16 * 16;
  std::vector<char> st_rec(staged ? (size_t)D * e_stride * st_rsb : 16, 0);
  if (staged)
    for (int d = 0; d < D; ++d)
      for (int pos = 0; pos < nc; ++pos) {
        const size_t at = (size_t)d * e_stride + pos;
        char *rec = &st_rec[at * st_rsb];
        double dv[3 + 7] = {0.0, Qdot ? Qdot[cellat[at]] : 0.0, gout[at]};
        int32_t uv[7];
        for (int k = 0; k < MI; ++k) {
          dv[3 + k] = gin[(size_t)k * D * e_stride + at];
          uv[k] = st_up[(size_t)k * D * e_stride + at];
        }
        std::memcpy(rec, dv, sizeof(double) * (3 + MI));
        std::memcpy(rec + sizeof(double) * (3 + MI), uv, sizeof(int32_t) * MI);
      }

  std::vector<int32_t> lvl_ptr((size_t)D * (l_max + 1), 0);
  for (int d = 0; d < D; ++d) {
    for (int l = 0; l <= l_max; ++l) lvl_ptr[(size_t)d * (l_max + 1) + l] = lvl_ptrs[d][std::min(l, n_lvl[d])];
  }
  std::vector<double> kA(B), kS(B), itau(B);
  for (int b = 0; b < B; ++b) {
    kA[b] = cm.C[b] / (cm.W * cm.tau[b]);
    kS[b] = cm.share[b] / cm.W;
    itau[b] = 1.0 / cm.tau[b];
  }
  std::vector<int32_t> dir_cls(D);
  std::iota(dir_cls.begin(), dir_cls.end(), 0);

  h->kind = 1; h->n_cells = nc; h->n_cls = D; h->n_planes = l_max; h->n_tasks = D * NBG;
  h->sweep_G = BG; h->sweep_threads = threads; h->sweep_rmax = MI; h->pencil_axis = -1;
  h->n_pos = nc; h->e_stride = e_stride; h->sweep_smem = (size_t)rcap * BG * sizeof(double);
  h->uns_staged = staged;
  if (staged) {
    h->sweep_smem = st_smem;
    h->n_tasks = D * st_NBG; h->sweep_G = st_BG; h->sweep_threads = st_threads;
  }
  h->T_ref = opt->T_ref;
  h->cg_rtol = opt->cg_rtol > 0 ? opt->cg_rtol : 1e-12;
  h->cg_max_iter = opt->cg_max_iter > 0 ? opt->cg_max_iter : 100000;
  if (!h->uns) h->uns = new (std::nothrow) UnsArgs();
  if (!h->uns) return nb_fail(h, NANOBTE_E_ALLOC, "host allocation failed");
  UnsArgs &u = *h->uns;

  for (int pass = 0; pass < 2; ++pass) {
    const bool dry = pass == 0;
    Arena A(h, dry);
    rc = nb_upload_generic(h, A, cm, G);
    if (rc) return nb_fail(h, rc, "device upload failed");
    u.D = D; u.B = B; u.BG = BG; u.NBG = NBG; u.MI = MI; u.cpp = cpp; u.rcap = rcap; u.n_act = nc; u.l_max = l_max; u.e_stride = e_stride;
    u.st_BG = st_BG; u.st_NBG = st_NBG; u.st_threads = st_threads; u.st_vr = st_vr; u.st_rr = st_rr; u.st_sr = st_sr;
    u.st_rec = A.put(st_rec);
    u.st_rsb = st_rsb;
    u.side_ptr = A.put(side_ptr);
    u.side_src = A.put(side_src);
    u.side_base = A.put(side_base);
    u.n_lvl = A.put(n_lvl);
    u.lvl_ptr = A.put(lvl_ptr);
    u.cell = A.put(cellat);
    u.up = A.put(up);
    u.gin = A.put(gin);
    u.gout = A.put(gout);
    u.kA = A.put(kA); u.kS = A.put(kS); u.itau = A.put(itau);
    u.vb = h->bd.v;
    u.theta = h->theta; u.Qdot = h->Qdot;
    u.bin = h->bd.bin; u.dir_bin = h->bd.dir_bin; u.dir_nin = h->bd.dir_nin;
    h->a2pos = A.put(a2pos);
    u.a2pos = h->a2pos;
    h->dir_cls = A.put(dir_cls);
    u.w = h->bd.w;
    u.s = A.put(cm.s);
    u.theta_SI = h->theta_SI; u.theta_en = h->theta_en; u.q = h->q;
    u.beta = cm.beta; u.Csum = cm.Csum;
    const size_t part_n = (size_t)3 * nc + 64;  // scratch of the host-destination getters
    h->part = A.zeros<double>(part_n);
    double *e = A.zeros<double>((size_t)D * e_stride * B);
    u.e = e; h->sw.e = e; h->bd.e = e; h->bd.e_stride = e_stride;
    if (A.rc) return nb_fail(h, A.rc, "device upload failed");
    if (dry) {
      const size_t need = A.off + 256;
      if (size_only) { *bytes_out = need; return 0; }
      if (opt->workspace) {
        if (opt->workspace_bytes < need) return nb_fail(h, NANOBTE_E_ALLOC, "workspace of %zu B given, %zu B needed", opt->workspace_bytes, need);
        if ((uintptr_t)opt->workspace & 255) return nb_fail(h, NANOBTE_E_INVALID, "workspace must be 256-byte aligned");
        h->arena = (char *)opt->workspace; h->arena_owned = false;
      } else {
        void *p = nullptr;
        if (cudaMalloc(&p, need) != cudaSuccess) { cudaGetLastError(); return nb_fail(h, NANOBTE_E_ALLOC, "cudaMalloc of %zu B failed", need); }
        h->arena = (char *)p; h->arena_owned = true;
      }
      h->arena_bytes = need;
    }
  }
  NB_CUDA(h, cudaMallocHost((void **)&h->h_pinned, 64));
  NB_CUDA(h, cudaStreamSynchronize(h->stream));  // host vectors die here
  rc = nb_launch_boundary(h, 1);  // initial inflow cache: thermalizing constants, zero elsewhere (R12)
  if (rc < 0) return rc;
  NB_CUDA(h, cudaStreamSynchronize(h->stream));
  return 0;
}

}  // namespace

extern "C" int nanobte_workspace_bytes_unstructured(const nanobte_unstructured_mesh *m, const nanobte_bands *b,
                                                    const nanobte_quadrature *q, const nanobte_tag *tags, int32_t n_tags,
                                                    const nanobte_options *opt, size_t *bytes_out) {
  if (!bytes_out) return NANOBTE_E_INVALID;
  nanobte_solver tmp;
  nb_query_sm_count(&tmp);
  int rc = build_uns(&tmp, m, b, q, tags, n_tags, nullptr, opt, true, bytes_out);
  nb_free_unstructured(&tmp);
  return rc;
}

extern "C" int nanobte_create_unstructured(const nanobte_unstructured_mesh *m, const nanobte_bands *b, const nanobte_quadrature *q,
                                           const nanobte_tag *tags, int32_t n_tags, const double *Qdot,
                                           const nanobte_options *opt, nanobte_solver **out) {
  if (!out) return NANOBTE_E_INVALID;
  nanobte_solver *h = new (std::nothrow) nanobte_solver();
  if (!h) return NANOBTE_E_ALLOC;
  *out = h;
  int rc = nb_check_device(h);
  if (rc) return rc;
  h->stream = opt ? (cudaStream_t)opt->stream : nullptr;
  rc = build_uns(h, m, b, q, tags, n_tags, Qdot, opt, false, nullptr);
  if (rc < 0 && h->arena && h->arena_owned) cudaFree(h->arena);
  if (rc < 0) h->arena = nullptr;
  return rc;
}
