// dao_master.cu -- step 8, the restricted master problem  min_{y >= 0} F(A y)
// by gradient projection, kept entirely on the device: ONE persistent cooperative kernel, one
// CTA per SM, each CTA owning a fixed slab of voxels (so its part of the dense aperture-dose
// block A stays in the L2 slice it was read from).  Per projected-gradient iteration:
//   G  z <- z + t dz, g = dF/dz on the slab (tile by tile through shared memory),
//      grad_k = a_k . g for every aperture k           -> one pass over A, one grid reduction
//   P  every CTA derives the same search direction p (projected steepest descent, optionally
//      with Polak-Ribiere+ conjugation on the free face) from the reduced gradient
//   D  dz = A p on the slab, curvature phi''(0)        -> one pass over A, one grid reduction
//   L  safeguarded Newton search for the root of phi'(t) = dz . g(z + t dz) on [0, t_max]
//                                                       -> passes over (z, dz) only
// The paper defers the step rule to Men et al. 2009 / Bazaraa et al.; the rule used
// here is DESIGN.md reading S2.  All reductions are fp64 and in a fixed order (bit-reproducible).
#include "dao_internal.cuh"

#include <math_constants.h>

namespace dao {

struct MasterParams {
  const float *A;
  int32_t n_vox_pad;
  const uint8_t *sid;
  const StructEntry *stab;
  double *mz;
  double *mdz;
  double *y;
  double *part;            // [grid][kMaxRedux]
  double *result;          // [kMaxRedux]
  DevState *st;
  dao_iter_record *history;
  const int32_t *ap_beam;
  int32_t add_candidate;
  int32_t max_iter;
  int32_t method;
  int32_t k_max;
  double tol;
};

constexpr double kLineSearchTol = 1e-4;   // |phi'(t)| <= kLineSearchTol * |phi'(0)| ends the line search

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t *p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u32(uint32_t *p, uint32_t v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_min_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Grid-wide sum of n (<= kMaxRedux) doubles: every CTA contributes vals[0..n), every CTA gets the
// totals in out[0..n).  The last CTA to arrive adds the per-CTA partials in CTA order, publishes
// the result and releases the others (sense = generation counter).  Requires co-resident CTAs
// (cooperative launch).
__device__ void grid_reduce(const MasterParams &p, int n, const double *vals, double *out) {
  __shared__ uint32_t s_gen;
  __shared__ int s_last;
  const int tid = threadIdx.x;
  double *mine = p.part + (size_t)blockIdx.x * kMaxRedux;
  if (tid < n) mine[tid] = vals[tid];
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    s_gen = ld_acquire_u32(&p.st->bar_gen);
    const uint32_t ticket = atomicAdd(&p.st->bar_count, 1u);
    s_last = (ticket == gridDim.x - 1);
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    // n_pad = n rounded up to a power of two <= blockDim; thread (i, part) adds the partials of the
    // CTAs b = part, part + P, ... in that order; the P parts of a value are then added in order.
    int n_pad = 1;
    while (n_pad < n) n_pad <<= 1;
    const int P = (int)blockDim.x / n_pad;          // >= 2 (n <= kMaxRedux <= blockDim/2)
    const int i = tid % n_pad, part = tid / n_pad;
    double s = 0.0;
    if (i < n && part < P) {
      for (unsigned b = part; b < gridDim.x; b += P) s += __ldcg(p.part + (size_t)b * kMaxRedux + i);
    }
    __shared__ double s_red[kMasterThreads];
    s_red[tid] = s;
    __syncthreads();
    if (tid < n) {
      double t = 0.0;
      for (int q = 0; q < P; ++q) t += s_red[q * n_pad + tid];
      p.result[tid] = t;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      p.st->bar_count = 0u;
      __threadfence();
      red_release_add_u32(&p.st->bar_gen, 1u);
    }
  } else {
    if (tid == 0) {
      while (ld_acquire_u32(&p.st->bar_gen) == s_gen) { __nanosleep(20); }
    }
  }
  __syncthreads();
  if (tid < n) out[tid] = __ldcg(p.result + tid);
  __syncthreads();
}

// Block-wide sums of NV per-thread doubles -> vals[0..NV) (fixed order: shuffle tree, then warps in order)
template <int NV>
__device__ void block_sum(double (&v)[NV], double *scratch /*[nwarps*NV]*/, double *vals) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const double s = warp_sum_d(v[i]);
    if (lane == 0) scratch[warp * NV + i] = s;
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double s = 0.0;
    for (int w = 0; w < nw; ++w) s += scratch[w * NV + threadIdx.x];
    vals[threadIdx.x] = s;
  }
  __syncthreads();
}

__global__ void __launch_bounds__(kMasterThreads, 1) k_master(MasterParams p) {
  // ---- shared state (replicated in every CTA, evolves identically everywhere) ----
  __shared__ double y_s[DAO_MAX_APERTURES];
  __shared__ double grad_s[kMaxRedux];
  __shared__ double pg_s[DAO_MAX_APERTURES];       // projected steepest descent of this iteration
  __shared__ double pgold_s[DAO_MAX_APERTURES];
  __shared__ double p_s[DAO_MAX_APERTURES];        // search direction (fp32-representable values)
  __shared__ double vals_s[kMaxRedux];
  __shared__ double red_s[kMaxRedux];
  __shared__ double g_tile[kMasterTile];
  // per-warp partials; aliases g_tile (only used once the tile loop of a phase is over)
  static_assert(kMasterTile >= (kMasterThreads / 32) * DAO_MAX_APERTURES, "warp_part must fit in g_tile");
  double *warp_part = g_tile;
  __shared__ StructEntry stab_s[256];
  __shared__ double sc[16];                        // broadcast scalars
  __shared__ int si[8];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = kMasterThreads / 32;
  const int K0 = p.st->K;
  const int cand = p.st->cand_valid;
  const int added = (p.add_candidate && cand) ? 1 : 0;
  const int K = K0 + added;
  if ((p.add_candidate && !added) || K == 0) {     // converged, pool full or empty pool: nothing to do
    if (blockIdx.x == 0 && tid == 0) { p.st->m_added = 0; p.st->m_iters = 0; }
    return;
  }

  for (int i = tid; i < 256; i += blockDim.x) stab_s[i] = p.stab[i];
  if (tid < DAO_MAX_APERTURES) {
    y_s[tid] = (tid < K0) ? p.y[tid] : 0.0;
    pgold_s[tid] = 0.0;
    p_s[tid] = 0.0;
  }
  __syncthreads();

  // slab of voxels owned by this CTA (multiple of 128 so that every warp strip is full)
  const int vpad = p.n_vox_pad;
  int slab = (vpad + (int)gridDim.x - 1) / (int)gridDim.x;
  slab = (slab + 127) / 128 * 128;
  const long long v0l = (long long)blockIdx.x * slab;
  const int v0 = (int)(v0l < vpad ? v0l : vpad);
  const int v1 = (v0 + slab < vpad) ? v0 + slab : vpad;

  // ---- z = A y on the slab (fp64), dz = 0 ----
  for (int v = v0 + tid * 4; v < v1; v += blockDim.x * 4) {
    double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
    for (int k = 0; k < K; ++k) {
      const double yk = y_s[k];
      if (yk == 0.0) continue;
      const float4 a = *reinterpret_cast<const float4 *>(p.A + (size_t)k * vpad + v);
      a0 = fma(yk, (double)a.x, a0); a1 = fma(yk, (double)a.y, a1);
      a2 = fma(yk, (double)a.z, a2); a3 = fma(yk, (double)a.w, a3);
    }
    p.mz[v] = a0; p.mz[v + 1] = a1; p.mz[v + 2] = a2; p.mz[v + 3] = a3;
    p.mdz[v] = 0.0; p.mdz[v + 1] = 0.0; p.mdz[v + 2] = 0.0; p.mdz[v + 3] = 0.0;
  }
  __syncthreads();

  double t_step = 0.0;          // step to apply to z at the start of the next G phase
  int iters = 0, restarts = 0, since_restart = 0;
  bool force_restart = true;
  unsigned free_prev[4] = {0u, 0u, 0u, 0u};
  int hit_max = 0;
  double F = 0.0, kkt = 0.0, pgmax = 0.0;

  for (;;) {
    // ================= phase G: z += t dz, g(z), grad = A^T g, F ==========================
    double accq[4] = {0.0, 0.0, 0.0, 0.0};   // lane l holds grad partials of k = q*32 + l (this warp's strips)
    double f_acc = 0.0;
    for (int tile0 = v0; tile0 < v1; tile0 += kMasterTile) {
      const int tn = (v1 - tile0 < kMasterTile) ? (v1 - tile0) : kMasterTile;
      for (int i = tid; i < tn; i += blockDim.x) {
        const int v = tile0 + i;
        double z = p.mz[v];
        if (t_step != 0.0) { z = fma(t_step, p.mdz[v], z); p.mz[v] = z; }
        const int s = p.sid[v];
        double gv = 0.0;
        if (s != kNoStruct) {
          const StructEntry e = stab_s[s];
          const double u = fmax(e.tm - z, 0.0), o = fmax(z - e.tp, 0.0);
          f_acc += e.a * u * u + e.b * o * o;
          gv = -2.0 * e.a * u + 2.0 * e.b * o;
        }
        g_tile[i] = gv;
      }
      __syncthreads();
      // warp `warp` owns the 128-voxel strips warp, warp+NW, ... of the tile; lane owns 4 voxels
      for (int s0 = warp * 128; s0 < tn; s0 += NW * 128) {
        const int vi = s0 + lane * 4;
        const double g0 = g_tile[vi], g1 = g_tile[vi + 1], g2 = g_tile[vi + 2], g3 = g_tile[vi + 3];
        const float *base = p.A + (size_t)(tile0 + vi);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int kq = q * 32;
          if (kq >= K) break;
          const int kn = (K - kq < 32) ? (K - kq) : 32;
          int l = 0;
          for (; l + 4 <= kn; l += 4) {
            float4 a[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
              a[u] = *reinterpret_cast<const float4 *>(base + (size_t)(kq + l + u) * vpad);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              double d = (double)a[u].x * g0;
              d = fma((double)a[u].y, g1, d);
              d = fma((double)a[u].z, g2, d);
              d = fma((double)a[u].w, g3, d);
              d = warp_sum_d(d);
              if (lane == l + u) accq[q] += d;
            }
          }
          for (; l < kn; ++l) {
            const float4 a = *reinterpret_cast<const float4 *>(base + (size_t)(kq + l) * vpad);
            double d = (double)a.x * g0;
            d = fma((double)a.y, g1, d);
            d = fma((double)a.z, g2, d);
            d = fma((double)a.w, g3, d);
            d = warp_sum_d(d);
            if (lane == l) accq[q] += d;
          }
        }
      }
      __syncthreads();
    }
    // combine the warps of the CTA in warp order
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int k = q * 32 + lane;
      if (k < K) warp_part[warp * DAO_MAX_APERTURES + k] = accq[q];
    }
    {
      const double fs = warp_sum_d(f_acc);
      if (lane == 0) red_s[warp] = fs;
    }
    __syncthreads();
    if (tid < K) {
      double s = 0.0;
      for (int w = 0; w < NW; ++w) s += warp_part[w * DAO_MAX_APERTURES + tid];
      vals_s[tid] = s;
    }
    if (tid == K) {
      double s = 0.0;
      for (int w = 0; w < NW; ++w) s += red_s[w];
      vals_s[K] = s;
    }
    __syncthreads();
    grid_reduce(p, K + 1, vals_s, grad_s /* K grads, then F */);
    if (tid == 0) sc[0] = grad_s[K];
    __syncthreads();
    F = sc[0];

    // ================= phase P: direction (warp 0, identical in every CTA) ================
    if (warp == 0) {
      double pg_max = 0.0, y_max = 1.0, kkt_l = 0.0, num = 0.0, den = 0.0;
      unsigned free_now[4] = {0u, 0u, 0u, 0u};
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int k = q * 32 + lane;
        bool fr = false;
        if (k < K) {
          const double gk = grad_s[k], yk = y_s[k];
          fr = (yk > 0.0) || (gk < 0.0);
          const double pgk = fr ? -gk : 0.0;
          pg_s[k] = pgk;
          pg_max = fmax(pg_max, fabs(pgk));
          y_max = fmax(y_max, yk);
          kkt_l = fmax(kkt_l, (yk > 0.0) ? fabs(gk) : fmax(-gk, 0.0));
          num += pgk * (pgk - pgold_s[k]);
          den += pgold_s[k] * pgold_s[k];
        }
        free_now[q] = __ballot_sync(0xffffffffu, fr);
      }
      pg_max = warp_max_d(pg_max);
      y_max = warp_max_d(y_max);
      kkt_l = warp_max_d(kkt_l);
      num = warp_sum_d(num);
      den = warp_sum_d(den);
      const bool conv = pg_max * y_max <= p.tol * fmax(F, 1e-300);
      const bool stop = conv || iters >= p.max_iter;
      bool same_free = true;
#pragma unroll
      for (int q = 0; q < 4; ++q) same_free = same_free && (free_now[q] == free_prev[q]);
      bool restart = force_restart || !same_free || p.method == 0 || since_restart >= K + 8 || !(den > 0.0);
      double beta = 0.0;
      if (!restart) beta = fmax(num / den, 0.0);
      if (beta == 0.0) restart = true;
      // direction, rounded to fp32-representable values
      double slope = 0.0;
      bool infeasible = false;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int k = q * 32 + lane;
        if (k < K) {
          double pk = pg_s[k];
          if (!restart && pk != 0.0) pk = fma(beta, p_s[k], pk);
          if (!restart && pg_s[k] == 0.0) pk = 0.0;
          pk = (double)(float)pk;
          if (pk < 0.0 && !(y_s[k] > 0.0)) infeasible = true;
          slope = fma(pk, grad_s[k], slope);
          vals_s[k] = pk;     // tentative
        }
      }
      slope = warp_sum_d(slope);
      infeasible = __any_sync(0xffffffffu, infeasible);
      if (!restart && (infeasible || !(slope < 0.0))) {
        restart = true;
        slope = 0.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int k = q * 32 + lane;
          if (k < K) {
            const double pk = (double)(float)pg_s[k];
            slope = fma(pk, grad_s[k], slope);
            vals_s[k] = pk;
          }
        }
        slope = warp_sum_d(slope);
      }
      double tmax = CUDART_INF;
      int kb = 0x7fffffff;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int k = q * 32 + lane;
        if (k < K) {
          const double pk = vals_s[k];
          p_s[k] = pk;
          pgold_s[k] = pg_s[k];
          if (pk < 0.0) {
            const double tk = y_s[k] / (-pk);
            if (tk < tmax) { tmax = tk; kb = k; }
          }
        }
      }
      {
        const double tmin = warp_min_d(tmax);
        const unsigned m = __ballot_sync(0xffffffffu, tmax == tmin && kb != 0x7fffffff);
        int kb_w = 0x7fffffff;
        if (m) {
          // smallest k among the lanes that attain the minimum
          int cand_k = (tmax == tmin) ? kb : 0x7fffffff;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) cand_k = min(cand_k, __shfl_xor_sync(0xffffffffu, cand_k, o));
          kb_w = cand_k;
        }
        tmax = tmin;
        kb = kb_w;
      }
      if (lane == 0) {
        sc[1] = slope; sc[2] = tmax; sc[3] = pg_max; sc[4] = kkt_l;
        si[0] = stop ? 1 : 0; si[1] = (stop && !conv) ? 1 : 0; si[2] = kb; si[3] = restart ? 1 : 0;
        si[4] = (!(slope < 0.0)) ? 1 : 0;
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) free_prev[q] = free_now[q];
    }
    __syncthreads();
    pgmax = sc[3];
    kkt = sc[4];
    if (si[0] || si[4]) { hit_max = si[1]; break; }   // converged, iteration cap, or no descent left
    const double slope0 = sc[1], tmax = sc[2];
    const int kb = si[2];
    if (si[3]) { ++restarts; since_restart = 0; } else { ++since_restart; }
    force_restart = false;

    // ================= phase D: dz = A p, curvature =======================================
    double h_acc = 0.0;
    for (int vb = v0 + warp * 128; vb < v1; vb += NW * 128) {
      const int v = vb + lane * 4;
      const float *base = p.A + (size_t)v;
      double d0 = 0, d1 = 0, d2 = 0, d3 = 0;
      int k = 0;
      for (; k + 4 <= K; k += 4) {
        float4 a[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) a[u] = *reinterpret_cast<const float4 *>(base + (size_t)(k + u) * vpad);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const double pk = p_s[k + u];
          d0 = fma(pk, (double)a[u].x, d0); d1 = fma(pk, (double)a[u].y, d1);
          d2 = fma(pk, (double)a[u].z, d2); d3 = fma(pk, (double)a[u].w, d3);
        }
      }
      for (; k < K; ++k) {
        const float4 a = *reinterpret_cast<const float4 *>(base + (size_t)k * vpad);
        const double pk = p_s[k];
        d0 = fma(pk, (double)a.x, d0); d1 = fma(pk, (double)a.y, d1);
        d2 = fma(pk, (double)a.z, d2); d3 = fma(pk, (double)a.w, d3);
      }
      const double dd[4] = {d0, d1, d2, d3};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        p.mdz[v + u] = dd[u];
        const int s = p.sid[v + u];
        if (s != kNoStruct) {
          const StructEntry e = stab_s[s];
          const double z = p.mz[v + u];
          const double c = (z < e.tm ? e.a : 0.0) + (z > e.tp ? e.b : 0.0);
          h_acc = fma(2.0 * c * dd[u], dd[u], h_acc);
        }
      }
    }
    {
      double hv[1] = {h_acc};
      block_sum<1>(hv, warp_part, vals_s);
    }
    grid_reduce(p, 1, vals_s, red_s);
    const double h0 = red_s[0];

    // ================= phase L: root of phi'(t) on [0, tmax] ==============================
    // phi' is non-decreasing and piecewise linear; phi'(0) = slope0 < 0.
    double lo = 0.0, slo = slope0, hi = CUDART_INF, shi = 0.0;
    double t = (h0 > 0.0) ? (-slope0 / h0) : ((tmax < CUDART_INF) ? tmax : 1.0);
    if (t > tmax) t = tmax;
    bool hit_bound = false;
    for (int ls = 0; ls < 40; ++ls) {
      double acc3[3] = {0.0, 0.0, 0.0};   // phi'(t), phi''(t), F(t)
      for (int v = v0 + tid; v < v1; v += blockDim.x) {
        const int s = p.sid[v];
        if (s == kNoStruct) continue;
        const StructEntry e = stab_s[s];
        const double dz = p.mdz[v];
        const double z = fma(t, dz, p.mz[v]);
        const double u = fmax(e.tm - z, 0.0), o = fmax(z - e.tp, 0.0);
        const double gv = -2.0 * e.a * u + 2.0 * e.b * o;
        const double c = (u > 0.0 ? e.a : 0.0) + (o > 0.0 ? e.b : 0.0);
        acc3[0] = fma(dz, gv, acc3[0]);
        acc3[1] = fma(2.0 * c * dz, dz, acc3[1]);
        acc3[2] += e.a * u * u + e.b * o * o;
      }
      block_sum<3>(acc3, warp_part, vals_s);
      grid_reduce(p, 3, vals_s, red_s);
      const double s1 = red_s[0], s2 = red_s[1];
      if (fabs(s1) <= kLineSearchTol * fabs(slope0)) break;      // exact enough
      double tn;
      if (s1 < 0.0) {
        if (t >= tmax) { hit_bound = true; break; }              // still descending at the bound
        lo = t; slo = s1;
        tn = (s2 > 0.0) ? t - s1 / s2 : 2.0 * t;
        if (hi < CUDART_INF && !(tn < hi)) tn = lo + (hi - lo) * (-slo) / (shi - slo);
        if (tn > tmax) tn = tmax;
      } else {
        hi = t; shi = s1;
        tn = (s2 > 0.0) ? t - s1 / s2 : 0.5 * (lo + hi);
        if (!(tn > lo)) tn = lo + (hi - lo) * (-slo) / (shi - slo);
      }
      if (!(tn > lo) || !(tn < hi)) tn = 0.5 * (lo + (hi < CUDART_INF ? hi : 2.0 * t));
      if (hi < CUDART_INF && (hi - lo) <= 1e-15 * hi) { t = (s1 < 0.0) ? hi : lo; if (t <= 0.0) t = hi; break; }
      if (tn == t) break;
      t = tn;
    }
    // ================= update y (every CTA identically); z is updated in the next G phase ==
    if (tid < K) {
      double yk = fma(t, p_s[tid], y_s[tid]);
      if (yk < 0.0) yk = 0.0;
      if (hit_bound && tid == kb) yk = 0.0;
      y_s[tid] = yk;
    }
    if (hit_bound) force_restart = true;
    t_step = t;
    ++iters;
    __syncthreads();
  }

  // ---- publish ----
  if (blockIdx.x == 0) {
    if (tid < K) p.y[tid] = y_s[tid];
    if (tid == 0) {
      DevState *st = p.st;
      st->K = K;
      st->m_iters = iters;
      st->m_hit_max = hit_max;
      st->m_restarts = restarts;
      st->m_added = added;
      st->m_F = F;
      st->m_kkt = kkt;
      st->m_pg = pgmax;
      st->pg_iter_total += iters;
      if (added) {
        st->cand_valid = 0;
        dao_iter_record rec;
        rec.k = K;
        rec.beam = p.ap_beam[K - 1];
        rec.n_pg_iter = iters;
        rec.duplicate = st->cand_dup;
        rec.price = st->cand_price;
        rec.objective_before = st->F;
        rec.objective = F;
        rec.kkt_residual = kkt;
        p.history[K - 1] = rec;
      }
    }
  }
}

cudaError_t master_configure(Ctx *c) {
  int nb = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_master, kMasterThreads, 0);
  if (e != cudaSuccess) return e;
  if (nb < 1) return cudaErrorLaunchOutOfResources;
  c->master_grid = c->n_sm;      // one CTA per SM
  return cudaSuccess;
}

cudaError_t launch_master(Ctx *c, bool add_candidate) {
  MasterParams p{};
  p.A = c->d.A;
  p.n_vox_pad = c->n_vox_pad;
  p.sid = c->d.sid;
  p.stab = c->d.stab;
  p.mz = c->d.mz;
  p.mdz = c->d.mdz;
  p.y = c->d.y;
  p.part = c->d.m_part;
  p.result = c->d.m_result;
  p.st = c->d.state;
  p.history = c->d.history;
  p.ap_beam = c->d.ap_beam;
  p.add_candidate = add_candidate ? 1 : 0;
  p.max_iter = c->opt.master_max_iter;
  p.method = c->opt.master_method;
  p.k_max = c->opt.k_max;
  p.tol = c->opt.master_tol;
  void *args[] = {&p};
  return cudaLaunchCooperativeKernel((void *)k_master, dim3(c->master_grid), dim3(kMasterThreads), args, 0,
                                     c->stream);
}

}  // namespace dao
