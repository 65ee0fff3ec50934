// dao_spmvt.cu -- step 4: w = D^T pi over the explicit CSR of D^T (eq. 8; the paper
// "computes the value placed in parentheses for each beamlet explicitly").  Rows = beamlets (~10^4
// entries each), entries = caller voxel ids in ascending order, so the voxels of a beamlet form
// runs of consecutive ids and the gather of pi (4 n_vox bytes, L2 resident, read through L1) touches
// few sectors.
//
// The entry array is cut into spans of kTChunk entries.  Persistent warps take spans from an atomic
// ticket counter (work stealing: any assignment gives the same numbers, every span has its own
// output slots).  A span inside one row (99 % of them) is reduced with 128-bit streaming loads and
// a shuffle tree; a span that straddles rows takes a warp-per-segment path.  k_spmvt_finish adds the
// slots of a row in span order: bit-reproducible, no floating-point atomics.
#include "dao_internal.cuh"
#include "dao_ptx.cuh"

#include <algorithm>

namespace dao {

__global__ void __launch_bounds__(kTThreads) k_spmvt(const int32_t *__restrict__ t_ptr,
                                                     const int32_t *__restrict__ t_row,
                                                     const float *__restrict__ t_val, int64_t nnz, int32_t n_spans,
                                                     const int32_t *__restrict__ first_row,
                                                     const int32_t *__restrict__ seg_base,
                                                     const float *__restrict__ g, double *__restrict__ segsum,
                                                     uint32_t *__restrict__ ticket,
                                                     const int32_t *__restrict__ skip) {
  const int lane = threadIdx.x & 31;
  if (skip && *skip) return;
  constexpr int kRound = 512;                       // entries per warp round: 4 x (int4 + float4) per lane
  for (;;) {
    int c = 0;
    if (lane == 0) c = (int)atomicAdd(ticket, 1u);
    c = __shfl_sync(0xffffffffu, c, 0);
    if (c >= n_spans) break;
    const int64_t cbeg = (int64_t)c * kTChunk;
    int64_t cend = cbeg + kTChunk;
    const bool full = cend <= nnz;
    if (!full) cend = nnz;
    const int first = first_row[c];
    const int sb = seg_base[c];
    const int nseg = seg_base[c + 1] - sb;
    if (nseg == 1 && full) {
      double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
      const int4 *pr = reinterpret_cast<const int4 *>(t_row + cbeg) + lane;
      const float4 *pv = reinterpret_cast<const float4 *>(t_val + cbeg) + lane;
#pragma unroll 1
      for (int r0 = 0; r0 < kTChunk / kRound; ++r0) {
        int4 rr[4];
        float4 vv[4];
#pragma unroll
        for (int it = 0; it < 4; ++it) {
          rr[it] = ld_stream_i32x4(pr + (r0 * 4 + it) * 32);
          vv[it] = ld_stream_f32x4(pv + (r0 * 4 + it) * 32);
        }
        float gg[16];
#pragma unroll
        for (int it = 0; it < 4; ++it) {
          gg[4 * it + 0] = ld_gather_f32(g + rr[it].x);
          gg[4 * it + 1] = ld_gather_f32(g + rr[it].y);
          gg[4 * it + 2] = ld_gather_f32(g + rr[it].z);
          gg[4 * it + 3] = ld_gather_f32(g + rr[it].w);
        }
        a0 = fma((double)vv[0].x, (double)gg[0], a0); a0 = fma((double)vv[0].y, (double)gg[1], a0);
        a0 = fma((double)vv[0].z, (double)gg[2], a0); a0 = fma((double)vv[0].w, (double)gg[3], a0);
        a1 = fma((double)vv[1].x, (double)gg[4], a1); a1 = fma((double)vv[1].y, (double)gg[5], a1);
        a1 = fma((double)vv[1].z, (double)gg[6], a1); a1 = fma((double)vv[1].w, (double)gg[7], a1);
        a2 = fma((double)vv[2].x, (double)gg[8], a2); a2 = fma((double)vv[2].y, (double)gg[9], a2);
        a2 = fma((double)vv[2].z, (double)gg[10], a2); a2 = fma((double)vv[2].w, (double)gg[11], a2);
        a3 = fma((double)vv[3].x, (double)gg[12], a3); a3 = fma((double)vv[3].y, (double)gg[13], a3);
        a3 = fma((double)vv[3].z, (double)gg[14], a3); a3 = fma((double)vv[3].w, (double)gg[15], a3);
      }
      double acc = (a0 + a1) + (a2 + a3);
      acc = warp_sum_f64(acc);
      if (lane == 0) segsum[sb] = acc;
    } else {
      for (int sgi = 0; sgi < nseg; ++sgi) {
        const int row = first + sgi;
        int64_t lo = t_ptr[row], hi = t_ptr[row + 1];
        if (lo < cbeg) lo = cbeg;
        if (hi > cend) hi = cend;
        double acc = 0.0;
        for (int64_t e = lo + lane; e < hi; e += 32) acc = fma((double)t_val[e], (double)__ldg(g + t_row[e]), acc);
        acc = warp_sum_f64(acc);
        if (lane == 0) segsum[sb + sgi] = acc;
      }
    }
  }
}

__global__ void k_spmvt_finish(int32_t n_bl, const int32_t *__restrict__ t_ptr,
                               const int32_t *__restrict__ first_row, const int32_t *__restrict__ seg_base,
                               const double *__restrict__ segsum, float *__restrict__ w,
                               uint32_t *__restrict__ ticket, const int32_t *__restrict__ skip) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (skip && *skip) return;
  if (i == 0) *ticket = 0u;                         // re-arm the span counter for the next launch
  if (i >= n_bl) return;
  const int64_t lo = t_ptr[i], hi = t_ptr[i + 1];
  double s = 0.0;
  if (hi > lo) {
    const int ca = (int)(lo / kTChunk), cb = (int)((hi - 1) / kTChunk);
    for (int c = ca; c <= cb; ++c) s += segsum[seg_base[c] + (i - first_row[c])];
  }
  w[i] = (float)s;
}

// Short beamlet rows (mean row length below one span, e.g. the paper's own problem sizes of a few hundred
// entries per beamlet): one warp per row of D^T, lanes stride over the row with 4
// independent accumulators, shuffle tree, w written directly -- no span tables, no second kernel.  Fixed
// order per row: bit-reproducible.
template <int WPR>   // warps per row: 1, 2, 4 or 8 (few rows -> more warps per row, so that the GPU is filled)
__global__ void __launch_bounds__(kTThreads) k_spmvt_rows(int32_t n_bl, const int32_t *__restrict__ t_ptr,
                                                          const int32_t *__restrict__ t_row,
                                                          const float *__restrict__ t_val, const float *__restrict__ g,
                                                          float *__restrict__ w, const int32_t *__restrict__ skip) {
  __shared__ double part[kTThreads / 32];
  if (skip && *skip) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int kRowsPerCta = (kTThreads / 32) / WPR;
  const int sub = warp % WPR;                         // this warp's share of the row
  for (int row0 = blockIdx.x * kRowsPerCta; row0 < n_bl; row0 += gridDim.x * kRowsPerCta) {
    const int row = row0 + warp / WPR;
    double acc = 0.0;
    if (row < n_bl) {
      const int lo = t_ptr[row], hi = t_ptr[row + 1];
      double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
      // the warps of a row interleave rounds of 128 entries
      for (int base = lo + 128 * sub; base < hi; base += 128 * WPR) {
        const int e = base + lane;
        if (base + 128 <= hi) {
          const int r0 = ld_stream_i32(t_row + e), r1 = ld_stream_i32(t_row + e + 32);
          const int r2 = ld_stream_i32(t_row + e + 64), r3 = ld_stream_i32(t_row + e + 96);
          const float v0 = ld_stream_f32(t_val + e), v1 = ld_stream_f32(t_val + e + 32);
          const float v2 = ld_stream_f32(t_val + e + 64), v3 = ld_stream_f32(t_val + e + 96);
          a0 = fma((double)v0, (double)ld_gather_f32(g + r0), a0);
          a1 = fma((double)v1, (double)ld_gather_f32(g + r1), a1);
          a2 = fma((double)v2, (double)ld_gather_f32(g + r2), a2);
          a3 = fma((double)v3, (double)ld_gather_f32(g + r3), a3);
        } else {
          for (int q = e; q < hi; q += 32)
            a0 = fma((double)ld_stream_f32(t_val + q), (double)ld_gather_f32(g + ld_stream_i32(t_row + q)), a0);
        }
      }
      acc = warp_sum_f64((a0 + a1) + (a2 + a3));
    }
    if (WPR == 1) {
      if (lane == 0 && row < n_bl) w[row] = (float)acc;
    } else {
      __syncthreads();
      if (lane == 0) part[warp] = acc;
      __syncthreads();
      if (sub == 0 && lane == 0 && row < n_bl) {
        double s = 0.0;
#pragma unroll
        for (int u = 0; u < WPR; ++u) s += part[warp + u];   // fixed order
        w[row] = (float)s;
      }
    }
  }
}

cudaError_t launch_spmv_t(Ctx *c, const float *g, float *w_out, const int32_t *skip) {
  if (c->n_bl > 0 && c->nnz / c->n_bl < kTChunk && !(c->opt.reserved & 4)) {
    const int wpb = kTThreads / 32;
    const int target = c->n_sm * 32;                  // warps that fill the GPU
    int wpr = 1;
    while (wpr < wpb && c->n_bl * wpr < target) wpr *= 2;
    const int rows_per_cta = wpb / wpr;
    const int grid = std::max(1, std::min((c->n_bl + rows_per_cta - 1) / rows_per_cta, c->n_sm * kTCtasPerSm));
    ++c->n_launches;
    switch (wpr) {
      case 1: k_spmvt_rows<1><<<grid, kTThreads, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_row, c->d.t_val, g, w_out, skip); break;
      case 2: k_spmvt_rows<2><<<grid, kTThreads, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_row, c->d.t_val, g, w_out, skip); break;
      case 4: k_spmvt_rows<4><<<grid, kTThreads, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_row, c->d.t_val, g, w_out, skip); break;
      default: k_spmvt_rows<8><<<grid, kTThreads, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_row, c->d.t_val, g, w_out, skip); break;
    }
    return cudaGetLastError();
  }
  if (c->n_tchunks > 0) {
    int grid = c->n_sm * kTCtasPerSm;
    const int need = (c->n_tchunks + kTThreads / 32 - 1) / (kTThreads / 32);
    if (grid > need) grid = need;
    ++c->n_launches;
    k_spmvt<<<grid, kTThreads, 0, c->stream>>>(c->d.t_ptr, c->d.t_row, c->d.t_val, c->nnz, c->n_tchunks,
                                               c->d.t_first_row, c->d.t_seg_base, g, c->d.t_segsum,
                                               &c->d.state->ticket_misc, skip);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  const int t = 128;
  ++c->n_launches;
  k_spmvt_finish<<<(c->n_bl + t - 1) / t, t, 0, c->stream>>>(c->n_bl, c->d.t_ptr, c->d.t_first_row,
                                                             c->d.t_seg_base, c->d.t_segsum, w_out,
                                                             &c->d.state->ticket_misc, skip);
  return cudaGetLastError();
}

}  // namespace dao
