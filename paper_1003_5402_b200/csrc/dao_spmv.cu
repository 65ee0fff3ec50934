// dao_spmv.cu -- the bandwidth-bound kernels of the hot path:
//   step 1  x_i = sum_{k : i in A_k} y_k                 (eq. 7)
//   step 2  z = D x over a sliced-ELL copy of D          (eq. 1)
//   step 3  F(z), pi = dF/dz fused into the epilogue     (PAPER.md:75-83 eq. 3-5, :246-254 eq. 9-10, :136)
//   step 4  w = D^T pi over an explicit CSR of D^T       (eq. 8)
//   step 7  a_K = D 1_A (same kernel as step 2)          (eq. 2)
#include "dao_internal.cuh"

namespace dao {

// streaming 32-bit loads that do not allocate in L1 (the matrix is read once per pass)
__device__ __forceinline__ int32_t ld_stream_i32(const int32_t *p) {
  int32_t v;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ float ld_stream_f32(const float *p) {
  float v;
  asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ int4 ld_stream_i32x4(const int4 *p) {
  int4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
               : "l"(p));
  return v;
}
__device__ __forceinline__ float4 ld_stream_f32x4(const float4 *p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(p));
  return v;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------
// step 1: beamlet intensities (eq. 7).  One thread per beamlet, apertures visited in pool order,
// fp64 accumulation, fp32 result.
// ------------------------------------------------------------------------------------------
__global__ void k_intensity(const DevState *__restrict__ st, int32_t n_bl, int32_t max_rows,
                            const int32_t *__restrict__ bl_row, const int32_t *__restrict__ row_beam,
                            const int32_t *__restrict__ beam_row_ptr, const int32_t *__restrict__ row_bl_ptr,
                            const int32_t *__restrict__ ap_beam, const int32_t *__restrict__ ap_left,
                            const int32_t *__restrict__ ap_right, const double *__restrict__ y,
                            float *__restrict__ x) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_bl) return;
  const int32_t K = st->K;
  const int32_t r = bl_row[i];
  const int32_t b = row_beam[r];
  const int32_t m = r - beam_row_ptr[b];
  const int32_t c = i - row_bl_ptr[r];
  double acc = 0.0;
  for (int32_t k = 0; k < K; ++k) {
    if (ap_beam[k] != b) continue;
    const int32_t l = ap_left[k * max_rows + m], rr = ap_right[k * max_rows + m];
    if (c >= l && c < rr) acc += y[k];
  }
  x[i] = (float)acc;
}

cudaError_t launch_intensity(Ctx *c) {
  const int t = 128;
  k_intensity<<<(c->n_bl + t - 1) / t, t, 0, c->stream>>>(c->d.state, c->n_bl, c->max_rows_per_beam,
                                                          c->d.bl_row, c->d.row_beam, c->d.beam_row_ptr,
                                                          c->d.row_bl_ptr, c->d.ap_beam, c->d.ap_left,
                                                          c->d.ap_right, c->d.y, c->d.x);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// steps 2, 3, 7: sliced-ELL SpMV.  A warp owns 32 consecutive internal rows = 32/C slices of C
// rows; lane -> (slice, row in slice).  Element k of a row sits at slice_off + k*C + row, so a
// warp-wide load touches 32/C fully used 4*C-byte segments.  Per-lane fp64 accumulation in the
// caller's column order (= ascending k), no cross-lane reduction.  Persistent grid: warps stride
// over the row groups.
// ------------------------------------------------------------------------------------------
struct SpmvParams {
  const int32_t *col;
  const float *val;
  const uint32_t *slice_off;
  const float *x;
  int32_t n_bl;
  int32_t n_groups;          // groups of 32 rows
  int32_t n_vox_pad;
  // outputs
  float *out;                // z (objective / plain) or the dose block A (column mode)
  float *g;
  const uint8_t *sid;
  const StructEntry *stab;
  const int32_t *perm;
  double *f_part;
  DevState *st;
};

template <int C, bool XS, int MODE>
__global__ void __launch_bounds__(kSpmvThreads, 2) k_spmv_sell(SpmvParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float *xs = reinterpret_cast<float *>(smem_raw);
  __shared__ double red[kSpmvThreads / 32];
  __shared__ StructEntry stab_s[MODE == kSpmvObjective ? 256 : 1];

  float *out = p.out;
  if (MODE == kSpmvColumn) {
    if (!p.st->cand_valid) return;                       // nothing to add (converged or pool full)
    out += (size_t)p.st->K * (size_t)p.n_vox_pad;
  }
  if (XS) {
    for (int i = threadIdx.x; i < p.n_bl; i += blockDim.x) xs[i] = p.x[i];
  }
  if (MODE == kSpmvObjective) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) stab_s[i] = p.stab[i];
  }
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int warps_per_block = blockDim.x >> 5;
  const int sub = lane / C;              // which slice of the group
  const int r = lane % C;                // row inside the slice
  constexpr int SPG = 32 / C;            // slices per group
  double f_acc = 0.0;

  for (int grp = blockIdx.x * warps_per_block + warp; grp < p.n_groups; grp += gridDim.x * warps_per_block) {
    const int slice = grp * SPG + sub;
    const uint32_t off = p.slice_off[slice];
    const int len = (int)((p.slice_off[slice + 1] - off) / C);
    const int32_t *pc = p.col + off + r;
    const float *pv = p.val + off + r;
    double acc = 0.0;
    int k = 0;
#pragma unroll 1
    for (; k + 8 <= len; k += 8) {
      int32_t cc[8];
      float vv[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        cc[u] = ld_stream_i32(pc + (k + u) * C);
        vv[u] = ld_stream_f32(pv + (k + u) * C);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const float xv = XS ? xs[cc[u]] : __ldg(p.x + cc[u]);
        acc = fma((double)vv[u], (double)xv, acc);
      }
    }
    for (; k < len; ++k) {
      const int32_t cc = ld_stream_i32(pc + k * C);
      const float vv = ld_stream_f32(pv + k * C);
      const float xv = XS ? xs[cc] : __ldg(p.x + cc);
      acc = fma((double)vv, (double)xv, acc);
    }
    const int i = grp * 32 + lane;       // internal row
    if (MODE == kSpmvObjective) {
      const int s = p.sid[i];
      double gv = 0.0;
      if (s != kNoStruct) {
        const StructEntry e = stab_s[s];
        const double u = fmax(e.tm - acc, 0.0);
        const double o = fmax(acc - e.tp, 0.0);
        f_acc += e.a * u * u + e.b * o * o;
        gv = -2.0 * e.a * u + 2.0 * e.b * o;
      }
      out[i] = (float)acc;
      p.g[i] = (float)gv;
    } else if (MODE == kSpmvPlainUserOrder) {
      const int32_t j = p.perm[i];
      if (j >= 0) out[j] = (float)acc;
    } else {
      out[i] = (float)acc;
    }
  }

  if (MODE == kSpmvObjective) {
    // block partial of F, then the last block to finish adds the partials in block order
    f_acc = warp_sum(f_acc);
    if (lane == 0) red[warp] = f_acc;
    __syncthreads();
    __shared__ bool is_last;
    if (threadIdx.x == 0) {
      double s = 0.0;
      for (int w = 0; w < warps_per_block; ++w) s += red[w];
      p.f_part[blockIdx.x] = s;
      __threadfence();
      const uint32_t t = atomicAdd(&p.st->ticket_spmv, 1u);
      is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last && warp == 0) {
      __threadfence();
      double s = 0.0;
      for (int b = lane; b < (int)gridDim.x; b += 32) s += __ldcg(p.f_part + b);
      s = warp_sum(s);
      if (lane == 0) {
        p.st->F = s;
        p.st->ticket_spmv = 0u;
      }
    }
  }
}

template <int MODE>
static cudaError_t launch_spmv_mode(Ctx *c, const float *x, float *out) {
  SpmvParams p{};
  p.col = c->d.sell_col;
  p.val = c->d.sell_val;
  p.slice_off = c->d.slice_off;
  p.x = x;
  p.n_bl = c->n_bl;
  p.n_groups = c->n_vox_pad / 32;
  p.n_vox_pad = c->n_vox_pad;
  p.out = out;
  p.g = c->d.g;
  p.sid = c->d.sid;
  p.stab = c->d.stab;
  p.perm = c->d.perm;
  p.f_part = c->d.f_part;
  p.st = c->d.state;
  const int groups_per_block = kSpmvThreads / 32;
  int grid = (p.n_groups + groups_per_block - 1) / groups_per_block;
  if (grid > c->spmv_grid) grid = c->spmv_grid;
  if (grid < 1) grid = 1;
  if (c->x_in_smem) {
    const size_t smem = (size_t)c->n_bl * sizeof(float);
    auto kern = k_spmv_sell<kSellC, true, MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kSpmvThreads, smem, c->stream>>>(p);
  } else {
    k_spmv_sell<kSellC, false, MODE><<<grid, kSpmvThreads, 0, c->stream>>>(p);
  }
  return cudaGetLastError();
}

cudaError_t launch_spmv(Ctx *c, SpmvMode mode, const float *x, float *out) {
  switch (mode) {
    case kSpmvObjective: return launch_spmv_mode<kSpmvObjective>(c, x, out);
    case kSpmvPlain: return launch_spmv_mode<kSpmvPlain>(c, x, out);
    case kSpmvColumn: return launch_spmv_mode<kSpmvColumn>(c, x, out);
    default: return launch_spmv_mode<kSpmvPlainUserOrder>(c, x, out);
  }
}

// ------------------------------------------------------------------------------------------
// step 4: w = D^T g over the explicit CSR of D^T (rows = beamlets, ~10^4 entries each).  The
// entry array is cut into chunks of kTChunk elements, one CTA per chunk.  A chunk that lies in
// one row (the common case) is reduced with 128-bit streaming loads; a chunk that straddles
// rows takes a generic warp-per-row-segment path.  Every (chunk, row) segment sum goes to its
// own slot; k_spmvt_finish adds the slots of a row in chunk order, so w is bit-reproducible
// without atomics.  g is gathered through L1/L2 (4 n_vox bytes, L2 resident).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kTThreads) k_spmvt(const int32_t *__restrict__ t_ptr,
                                                     const int32_t *__restrict__ t_row,
                                                     const float *__restrict__ t_val, int64_t nnz,
                                                     const int32_t *__restrict__ first_row,
                                                     const int32_t *__restrict__ seg_base,
                                                     const float *__restrict__ g, double *__restrict__ segsum) {
  __shared__ double red[kTThreads / 32];
  const int c = blockIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t cbeg = (int64_t)c * kTChunk;
  int64_t cend = cbeg + kTChunk;
  const bool full = cend <= nnz;
  if (!full) cend = nnz;
  const int first = first_row[c];
  const int nseg = seg_base[c + 1] - seg_base[c];
  if (nseg == 1 && full) {
    double acc = 0.0;
    const int4 *pr = reinterpret_cast<const int4 *>(t_row + cbeg);
    const float4 *pv = reinterpret_cast<const float4 *>(t_val + cbeg);
    constexpr int IT = kTChunk / (4 * kTThreads);
    int4 rr[IT];
    float4 vv[IT];
#pragma unroll
    for (int it = 0; it < IT; ++it) {
      rr[it] = ld_stream_i32x4(pr + it * kTThreads + threadIdx.x);
      vv[it] = ld_stream_f32x4(pv + it * kTThreads + threadIdx.x);
    }
#pragma unroll
    for (int it = 0; it < IT; ++it) {
      const float g0 = __ldg(g + rr[it].x), g1 = __ldg(g + rr[it].y);
      const float g2 = __ldg(g + rr[it].z), g3 = __ldg(g + rr[it].w);
      acc = fma((double)vv[it].x, (double)g0, acc);
      acc = fma((double)vv[it].y, (double)g1, acc);
      acc = fma((double)vv[it].z, (double)g2, acc);
      acc = fma((double)vv[it].w, (double)g3, acc);
    }
    acc = warp_sum(acc);
    if (lane == 0) red[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < kTThreads / 32; ++w) s += red[w];
      segsum[seg_base[c]] = s;
    }
  } else {
    for (int sgi = warp; sgi < nseg; sgi += kTThreads / 32) {
      const int row = first + sgi;
      int64_t lo = t_ptr[row], hi = t_ptr[row + 1];
      if (lo < cbeg) lo = cbeg;
      if (hi > cend) hi = cend;
      double acc = 0.0;
      for (int64_t e = lo + lane; e < hi; e += 32) acc = fma((double)t_val[e], (double)__ldg(g + t_row[e]), acc);
      acc = warp_sum(acc);
      if (lane == 0) segsum[seg_base[c] + sgi] = acc;
    }
  }
}

__global__ void k_spmvt_finish(int32_t n_bl, const int32_t *__restrict__ t_ptr,
                               const int32_t *__restrict__ first_row, const int32_t *__restrict__ seg_base,
                               const double *__restrict__ segsum, float *__restrict__ w) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_bl) return;
  const int64_t lo = t_ptr[i], hi = t_ptr[i + 1];
  double s = 0.0;
  if (hi > lo) {
    const int ca = (int)(lo / kTChunk), cb = (int)((hi - 1) / kTChunk);
    for (int c = ca; c <= cb; ++c) s += segsum[seg_base[c] + (i - first_row[c])];
  }
  w[i] = (float)s;
}

cudaError_t launch_spmv_t(Ctx *c, const float *g, float *w_out) {
  if (c->n_tchunks > 0) {
    k_spmvt<<<c->n_tchunks, kTThreads, 0, c->stream>>>(c->d.t_ptr, c->d.t_row, c->d.t_val, c->nnz,
                                                        c->d.t_first_row, c->d.t_seg_base, g, c->d.t_segsum);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  const int t = 128;
  k_spmvt_finish<<<(c->n_bl + t - 1) / t, t, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_first_row,
                                                             c->d.t_seg_base, c->d.t_segsum, w_out);
  return cudaGetLastError();
}

}  // namespace dao
