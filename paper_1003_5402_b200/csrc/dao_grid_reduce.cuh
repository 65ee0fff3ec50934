// dao_grid_reduce.cuh -- grid-wide fp64 reductions of the persistent master kernels (dao_master.cu,
// dao_newton.cu).  The data travel in flagged 16-byte slots ({lo32, epoch, hi32, epoch}): a reader
// polls the data itself, there is no counter and no separate release/acquire hop.  Small reductions
// (<= 16 values) are one hop (every CTA reads every CTA's slot); large ones are two hops (CTA i sums
// the values i, i + grid, ... over the grid in CTA order and publishes the totals).  All sums are
// fp64 in a fixed order: bit-reproducible and identical in every CTA.
#pragma once

#include "dao_internal.cuh"
#include "dao_ptx.cuh"

namespace dao {

constexpr int kNW = kMasterWorkers / 32;  // worker warps of the master kernels

// barrier over the worker warps only (the producer warp never joins it)
__device__ __forceinline__ void wsync() { asm volatile("bar.sync 1, %0;" ::"n"(kMasterWorkers) : "memory"); }

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
__device__ __forceinline__ unsigned long long gtimer() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// ---- flagged slots ---------------------------------------------------------------------------
__device__ __forceinline__ void ll_store(uint4 *slot, double v, uint32_t ep) {
  const unsigned long long u = (unsigned long long)__double_as_longlong(v);
  asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(slot), "r"((uint32_t)u), "r"(ep),
               "r"((uint32_t)(u >> 32)), "r"(ep)
               : "memory");
}
__device__ __forceinline__ uint4 ll_load(const uint4 *slot) {
  uint4 w;
  asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w)
               : "l"(slot)
               : "memory");
  return w;
}
__device__ __forceinline__ double ll_value(const uint4 &w) {
  return __longlong_as_double((long long)(((unsigned long long)w.z << 32) | (unsigned long long)w.x));
}

// One warp sums value `i` of every CTA's slot of this epoch: lane l takes the CTAs l, l+32, ...
// in that order, then a shuffle tree (fixed order).  Every lane returns the total.
// (A push variant -- every CTA stores into a private inbox of every reader -- was measured slower:
// 3.8 us against 2.6 us for the small reduction on B200.)
constexpr int kMaxGridOver32 = (kMasterMaxGrid + 31) / 32;
__device__ __forceinline__ double ll_warp_gather(const uint4 *part /*[grid][stride]*/, int stride, int i, uint32_t ep,
                                                 int lane) {
  const int grid = (int)gridDim.x;
  uint4 w[kMaxGridOver32];
#pragma unroll
  for (int j = 0; j < kMaxGridOver32; ++j) {
    const int b = lane + 32 * j;
    if (b < grid) w[j] = ll_load(part + (size_t)b * stride + i);
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < kMaxGridOver32; ++j) {
    const int b = lane + 32 * j;
    if (b < grid) {
      while (w[j].y != ep || w[j].w != ep) w[j] = ll_load(part + (size_t)b * stride + i);
      s += ll_value(w[j]);
    }
  }
  return warp_sum_f64(s);
}

struct Reducer {
  uint4 *part;      // [2][grid][stride]
  uint4 *result;    // [2][stride]
  uint32_t ep;      // epoch of the last reduction
  int stride;       // slots per CTA (>= the largest n ever reduced)

  // n <= kNW values: every CTA reads every CTA's slot (one hop).  vals/out in shared memory.
  __device__ __noinline__ void small(int n, const double *vals, double *out) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    ++ep;
    uint4 *buf = part + (size_t)(ep & 1u) * gridDim.x * stride;
    if (tid < n) ll_store(buf + (size_t)blockIdx.x * stride + tid, vals[tid], ep);
    if (warp < n) {
      const double s = ll_warp_gather(buf, stride, warp, ep, lane);
      if (lane == 0) out[warp] = s;
    }
    wsync();
  }
  // n <= stride values: CTA i sums the values i, i + grid, ... and publishes the totals (two hops).
  // vals and out may be the same array.
  __device__ __noinline__ void large(int n, const double *vals, double *out) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    ++ep;
    uint4 *buf = part + (size_t)(ep & 1u) * gridDim.x * stride;
    uint4 *res = result + (size_t)(ep & 1u) * stride;
    for (int i = tid; i < n; i += kMasterWorkers) ll_store(buf + (size_t)blockIdx.x * stride + i, vals[i], ep);
    // values this CTA owns: i = blockIdx.x + j * gridDim.x, one warp each
    for (int i = (int)blockIdx.x + warp * (int)gridDim.x; i < n; i += kNW * (int)gridDim.x) {
      const double s = ll_warp_gather(buf, stride, i, ep, lane);
      if (lane == 0) ll_store(res + i, s, ep);
    }
    for (int i = tid; i < n; i += kMasterWorkers) {
      uint4 w = ll_load(res + i);
      while (w.y != ep || w.w != ep) w = ll_load(res + i);
      out[i] = ll_value(w);
    }
    wsync();
  }
  // Same result as large() for many values (the Hessian of the Newton master): CTA c owns the CONTIGUOUS range
  // [c m, (c + 1) m), m = ceil(n / grid), so that what it gathers from every other CTA is one contiguous run of
  // slots (coalesced) instead of m scattered ones.  Warp w sums the sources w, w + 16, ... in that order, then
  // the warps are added in order.  scratch: >= kNW * m doubles of shared memory.  vals and out may alias.
  __device__ __noinline__ void ranges(int n, const double *vals, double *out, double *scratch) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grid = (int)gridDim.x;
    ++ep;
    uint4 *buf = part + (size_t)(ep & 1u) * grid * stride;
    uint4 *res = result + (size_t)(ep & 1u) * stride;
    for (int i = tid; i < n; i += kMasterWorkers) ll_store(buf + (size_t)blockIdx.x * stride + i, vals[i], ep);
    const int m = (n + grid - 1) / grid;
    const int lo = (int)blockIdx.x * m;
    const int cnt = max(0, min(m, n - lo));
    for (int l0 = 0; l0 < cnt; l0 += 32) {
      const int l = l0 + lane;
      if (l < cnt) {
        double s = 0.0;
        const uint4 *src = buf + lo + l;
        for (int b0 = warp; b0 < grid; b0 += kNW * 5) {
          uint4 w[5];
#pragma unroll
          for (int j = 0; j < 5; ++j) {
            const int b = b0 + j * kNW;
            if (b < grid) w[j] = ll_load(src + (size_t)b * stride);
          }
#pragma unroll
          for (int j = 0; j < 5; ++j) {
            const int b = b0 + j * kNW;
            if (b < grid) {
              while (w[j].y != ep || w[j].w != ep) w[j] = ll_load(src + (size_t)b * stride);
              s += ll_value(w[j]);
            }
          }
        }
        scratch[warp * m + l] = s;
      }
    }
    wsync();
    for (int l = tid; l < cnt; l += kMasterWorkers) {
      double t = 0.0;
      for (int w = 0; w < kNW; ++w) t += scratch[w * m + l];
      ll_store(res + lo + l, t, ep);
    }
    for (int i = tid; i < n; i += kMasterWorkers) {
      uint4 w = ll_load(res + i);
      while (w.y != ep || w.w != ep) w = ll_load(res + i);
      out[i] = ll_value(w);
    }
    wsync();
  }
};

// ---- the A stream of the master kernels: ring position, mbarrier helpers --------------------------
struct RingPos {
  int stage;
  uint32_t phase;
  __device__ __forceinline__ void advance(int n_stages) {
    if (++stage == n_stages) { stage = 0; phase ^= 1u; }
  }
};

__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_addr(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// non-blocking test (mbarrier.try_wait may suspend the thread up to a system time limit, ~0.5 us measured on B200,
// when the phase is not complete yet: never use it for "is it free?" checks)
__device__ __forceinline__ bool mbar_test_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_addr(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_spin_wait(uint64_t *bar, uint32_t parity) {
  while (!mbar_test_wait(bar, parity)) {}
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}

}  // namespace dao
