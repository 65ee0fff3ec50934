// dao_spmv.cu -- steps 1, 2, 3, 7 of the hot path:
//   step 1  x_i = sum_{k : i in A_k} y_k                 (eq. 7)
//   step 2  z = D x over a sliced-ELL copy of D          (eq. 1)
//   step 3  F(z), pi = dF/dz fused into the epilogue     (PAPER.md:75-83 eq. 3-5, :246-254 eq. 9-10, :136)
//   step 7  a_K = D 1_A (same kernel as step 2)          (eq. 2)
#include "dao_internal.cuh"
#include "dao_ptx.cuh"

namespace dao {

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
  if (c->x_current) return cudaSuccess;   // the master kernel already wrote x for this y
  const int t = 128;
  ++c->n_launches;
  k_intensity<<<(c->n_bl + t - 1) / t, t, 0, c->stream>>>(c->d.state, c->n_bl, c->max_rows_per_beam,
                                                          c->d.bl_row, c->d.row_beam, c->d.beam_row_ptr,
                                                          c->d.row_bl_ptr, c->d.ap_beam, c->d.ap_left,
                                                          c->d.ap_right, c->d.y, c->d.x);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// steps 2, 3, 7: sliced-ELL SpMV.  A warp owns one slice of 32 consecutive internal rows, lane =
// row; element k of a row sits at slice_off + 32 k + lane, so every warp-wide access is one fully
// used 128-byte line.  Per-lane fp64 accumulation in the caller's column order (= ascending k, the
// order of the oracle's row loop), no cross-lane reduction.  Persistent grid: warps stride over
// the slices.
// ------------------------------------------------------------------------------------------
struct SpmvParams {
  const int32_t *col;
  const float *val;
  const uint32_t *slice_off;
  const float *x;
  int32_t n_bl;
  int32_t n_slices;          // slices of 32 rows
  int32_t n_vox_pad;
  // outputs
  float *out;                // z (objective / plain) or the dose block A (column mode)
  float *g;
  const uint8_t *sid;
  const StructEntry *stab;
  const float *vt;           // per-voxel thresholds (re-optimisation mode) or null
  const int32_t *perm;
  double *f_part;
  DevState *st;
  const int32_t *skip;       // device flag (may be null): non-zero -> the launch does nothing
  // column mode: layout of the dose block A (a_index) and the column to write (< 0: the pool size K)
  int32_t a_T, a_TP, a_col, a_ntiles;
  int64_t a_stride;
  // column mode with a_col < 0: x is the 0/1 mask of the pending candidate, built while x is staged (no mask array,
  // no extra pass): beamlet i is open iff its leaf row belongs to the candidate's beam and i lies in [left, right)
  const int32_t *bl_row, *row_beam, *row_bl_ptr, *left, *right;
  int32_t mask_from_candidate;
};

template <int MODE>
__device__ __forceinline__ float spmv_x_of(const SpmvParams &p, int i, int cand_beam) {
  if (MODE == kSpmvColumn && p.mask_from_candidate) {
    const int32_t r = p.bl_row[i];
    if (p.row_beam[r] != cand_beam) return 0.f;
    const int32_t c = i - p.row_bl_ptr[r];
    return (c >= p.left[r] && c < p.right[r]) ? 1.f : 0.f;
  }
  return p.x[i];
}

// per-row epilogue: objective / gradient (step 3) or plain store
template <int MODE>
__device__ __forceinline__ void spmv_store(const SpmvParams &p, float *out, const StructEntry *stab_s, int i,
                                           double acc, double &f_acc, int kcol) {
  if (MODE == kSpmvObjective) {
    const int s = p.sid[i];
    double gv = 0.0;
    if (s != kNoStruct) {
      StructEntry e = stab_s[s];
      if (p.vt) e.tm = e.tp = (double)p.vt[i];       // T_j of eq. 3-4
      const double u = fmax(e.tm - acc, 0.0);
      const double o = fmax(acc - e.tp, 0.0);
      f_acc += e.a * u * u + e.b * o * o;
      gv = -2.0 * e.a * u + 2.0 * e.b * o;
    }
    const int32_t j = p.perm[i];         // z and pi are kept in the caller's voxel order
    if (j >= 0) {
      out[j] = (float)acc;
      p.g[j] = (float)gv;
    }
  } else if (MODE == kSpmvPlainUserOrder) {
    const int32_t j = p.perm[i];
    if (j >= 0) out[j] = (float)acc;
  } else if (MODE == kSpmvColumn) {
    out[a_index(p.a_T, p.a_TP, p.a_stride, p.n_vox_pad, p.a_ntiles, i, kcol)] = (float)acc;
  } else {
    out[i] = (float)acc;
  }
}

// block partial of F, then the last block to finish adds the partials in block order
__device__ __forceinline__ void spmv_finish_objective(const SpmvParams &p, double f_acc, double *red /*[nwarps]*/) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __shared__ bool is_last;
  f_acc = warp_sum_f64(f_acc);
  if (lane == 0) red[warp] = f_acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < nw; ++w) s += red[w];
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
    s = warp_sum_f64(s);
    if (lane == 0) {
      p.st->F = s;
      p.st->ticket_spmv = 0u;
    }
  }
}

// ---- variant A: the matrix streams through a warp-private cp.async.bulk (TMA) ring ---------------
// Every warp keeps kRingStages chunks of kRingK k-steps (kRingK * 32 * 8 bytes) in flight into its
// own shared-memory ring, completion signalled on per-stage mbarriers; lane 0 is the producer, the
// whole warp consumes.  Bytes in flight per SM = warps * stages * 4 KB, independent of registers.
constexpr int kRingK = 16;                                   // k-steps per chunk
constexpr int kRingStages = 3;
constexpr int kRingChunkElems = kRingK * 32;                 // per array
constexpr int kRingStageBytes = kRingChunkElems * 8;         // col + val

struct RingCursor {          // position in a warp's list of chunks
  int slice;                 // current slice (strided over the grid)
  int k0;                    // first k-step of the next chunk in that slice
  uint32_t off;              // slice_off[slice]
  int len;                   // k-steps of the slice
};

template <int MODE>
__global__ void __launch_bounds__(kSpmvRingThreads, 1) k_spmv_ring(SpmvParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int nw = blockDim.x >> 5;
  // layout: ring [nw][stages][col chunk | val chunk], barriers, x
  unsigned char *ring = smem_raw;
  uint64_t *bars = reinterpret_cast<uint64_t *>(ring + (size_t)nw * kRingStages * kRingStageBytes);
  float *xs = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(bars) + align_up_c(nw * kRingStages * 8, 128));
  __shared__ double red[kSpmvRingThreads / 32];
  __shared__ StructEntry stab_s[MODE == kSpmvObjective ? 256 : 1];

  float *out = p.out;
  if (p.skip && *p.skip) return;
  int kcol = 0;
  if (MODE == kSpmvColumn) {
    kcol = p.a_col;
    if (kcol < 0) {
      if (!p.st->cand_valid) return;                     // nothing to add (converged or pool full)
      kcol = p.st->K;
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
    for (int s = 0; s < kRingStages; ++s) mbar_init(&bars[warp * kRingStages + s], 1);
  }
  fence_mbar_init();
  __syncwarp();                 // the ring is warp-private: its first copies go out before x is staged

  const int stride = gridDim.x * nw;
  const int first = blockIdx.x * nw + warp;
  unsigned char *my_ring = ring + (size_t)warp * kRingStages * kRingStageBytes;
  uint64_t *my_bars = bars + warp * kRingStages;

  // producer cursor: skips empty slices
  RingCursor pc;
  pc.slice = first; pc.k0 = 0; pc.off = 0; pc.len = 0;
  auto load_slice = [&](RingCursor &c) {
    while (c.slice < p.n_slices) {
      const uint32_t o = p.slice_off[c.slice];
      const int len = (int)((p.slice_off[c.slice + 1] - o) >> 5);
      if (len > 0) { c.off = o; c.len = len; c.k0 = 0; return; }
      c.slice += stride;
    }
    c.len = 0;
  };
  load_slice(pc);
  uint32_t n_issued = 0, n_consumed = 0;
  auto issue = [&]() {                       // issue the chunk at the producer cursor (all lanes track it)
    if (pc.slice >= p.n_slices) return;
    const int kn = min(kRingK, pc.len - pc.k0);
    const uint32_t bytes = (uint32_t)kn * 32u * 4u;
    const int stage = n_issued % kRingStages;
    if (lane == 0) {
      unsigned char *dst = my_ring + (size_t)stage * kRingStageBytes;
      const size_t e0 = (size_t)pc.off + (size_t)pc.k0 * 32;
      mbar_arrive_expect_tx(&my_bars[stage], 2u * bytes);
      bulk_g2s(dst, p.col + e0, bytes, &my_bars[stage]);
      bulk_g2s(dst + kRingChunkElems * 4, p.val + e0, bytes, &my_bars[stage]);
    }
    ++n_issued;
    pc.k0 += kn;
    if (pc.k0 >= pc.len) { pc.slice += stride; load_slice(pc); }
  };
#pragma unroll
  for (int s = 0; s < kRingStages; ++s) issue();

  // x and the penalty table are staged while the first chunks are in flight
  {
    const int cand_beam = (MODE == kSpmvColumn && p.mask_from_candidate) ? p.st->cand_beam : 0;
    for (int i = threadIdx.x; i < p.n_bl; i += blockDim.x) xs[i] = spmv_x_of<MODE>(p, i, cand_beam);
  }
  if (MODE == kSpmvObjective) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) stab_s[i] = p.stab[i];
  }
  __syncthreads();

  double f_acc = 0.0;
  for (int slice = first; slice < p.n_slices; slice += stride) {
    const uint32_t off = p.slice_off[slice];
    const int len = (int)((p.slice_off[slice + 1] - off) >> 5);
    double acc = 0.0;
    for (int k0 = 0; k0 < len; k0 += kRingK) {
      const int kn = min(kRingK, len - k0);
      const int stage = n_consumed % kRingStages;
      mbar_wait(&my_bars[stage], (n_consumed / kRingStages) & 1u);
      const int32_t *sc = reinterpret_cast<const int32_t *>(my_ring + (size_t)stage * kRingStageBytes) + lane;
      const float *sv = reinterpret_cast<const float *>(my_ring + (size_t)stage * kRingStageBytes + kRingChunkElems * 4) + lane;
      if (kn == kRingK) {
#pragma unroll
        for (int k = 0; k < kRingK; ++k) acc = fma((double)sv[k * 32], (double)xs[sc[k * 32]], acc);
      } else {
        for (int k = 0; k < kn; ++k) acc = fma((double)sv[k * 32], (double)xs[sc[k * 32]], acc);
      }
      ++n_consumed;
      // every lane is done with the stage before it is refilled; the proxy fence orders the lanes' generic-proxy
      // reads before the bulk copy (async proxy) -- without it a refill was seen to overtake reads still queued
      // (k_spmvt_ring, where the values are consumed after the refill is issued)
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      issue();
    }
    spmv_store<MODE>(p, out, stab_s, slice * 32 + lane, acc, f_acc, kcol);
  }
  if (MODE == kSpmvObjective) spmv_finish_objective(p, f_acc, red);
}

// ---- variant B: direct global loads (used when x does not fit next to the ring) -------------------
template <bool XS, int MODE>
__global__ void __launch_bounds__(kSpmvThreads, 2) k_spmv_sell(SpmvParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float *xs = reinterpret_cast<float *>(smem_raw);
  __shared__ double red[kSpmvThreads / 32];
  __shared__ StructEntry stab_s[MODE == kSpmvObjective ? 256 : 1];

  float *out = p.out;
  if (p.skip && *p.skip) return;
  int kcol = 0;
  if (MODE == kSpmvColumn) {
    kcol = p.a_col;
    if (kcol < 0) {
      if (!p.st->cand_valid) return;                     // nothing to add (converged or pool full)
      kcol = p.st->K;
    }
  }
  if (XS) {
    const int cand_beam = (MODE == kSpmvColumn && p.mask_from_candidate) ? p.st->cand_beam : 0;
    for (int i = threadIdx.x; i < p.n_bl; i += blockDim.x) xs[i] = spmv_x_of<MODE>(p, i, cand_beam);
  }
  if (MODE == kSpmvObjective) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) stab_s[i] = p.stab[i];
  }
  __syncthreads();

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  double f_acc = 0.0;
  for (int slice = blockIdx.x * nw + warp; slice < p.n_slices; slice += gridDim.x * nw) {
    const uint32_t off = p.slice_off[slice];
    const int len = (int)((p.slice_off[slice + 1] - off) >> 5);
    const int32_t *pc = p.col + off + lane;
    const float *pv = p.val + off + lane;
    double acc = 0.0;
    int k = 0;
#pragma unroll 1
    for (; k + 8 <= len; k += 8) {
      int32_t cc[8];
      float vv[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        cc[u] = ld_stream_i32(pc + (k + u) * 32);
        vv[u] = ld_stream_f32(pv + (k + u) * 32);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const float xv = XS ? xs[cc[u]] : __ldg(p.x + cc[u]);
        acc = fma((double)vv[u], (double)xv, acc);
      }
    }
    for (; k < len; ++k) {
      const int32_t cc = ld_stream_i32(pc + k * 32);
      const float vv = ld_stream_f32(pv + k * 32);
      const float xv = XS ? xs[cc] : __ldg(p.x + cc);
      acc = fma((double)vv, (double)xv, acc);
    }
    spmv_store<MODE>(p, out, stab_s, slice * 32 + lane, acc, f_acc, kcol);
  }
  if (MODE == kSpmvObjective) spmv_finish_objective(p, f_acc, red);
}

template <int MODE>
static cudaError_t launch_spmv_mode(Ctx *c, const float *x, float *out, const int32_t *skip, int32_t a_col) {
  SpmvParams p{};
  p.col = c->d.sell_col;
  p.val = c->d.sell_val;
  p.slice_off = c->d.slice_off;
  p.x = x;
  p.n_bl = c->n_bl;
  p.n_slices = c->n_slices;
  p.n_vox_pad = c->n_vox_pad;
  p.out = out;
  p.g = c->d.g;
  p.sid = c->d.sid;
  p.vt = c->has_vt ? c->d.vt : nullptr;
  p.stab = c->d.stab;
  p.perm = c->d.perm;
  p.f_part = c->d.f_part;
  p.st = c->d.state;
  p.skip = skip;
  p.a_T = c->nwt.T; p.a_TP = c->nwt.TP; p.a_stride = c->nwt.tile_stride; p.a_col = a_col; p.a_ntiles = c->nwt.n_tiles;
  if (MODE == kSpmvColumn) p.out = c->d.A + (size_t)c->nwt.meta_rows * (size_t)c->nwt.TP;   // column 0 of tile 0
  p.bl_row = c->d.bl_row; p.row_beam = c->d.row_beam; p.row_bl_ptr = c->d.row_bl_ptr; p.left = c->d.left; p.right = c->d.right;
  p.mask_from_candidate = (MODE == kSpmvColumn && a_col < 0 && spmv_builds_mask(c)) ? 1 : 0;
  ++c->n_launches;
  if (c->spmv_ring_warps > 0) {
    const int nw = c->spmv_ring_warps;
    const size_t smem = (size_t)nw * kRingStages * kRingStageBytes + align_up((size_t)nw * kRingStages * 8, 128) +
                        align_up((size_t)c->n_bl * 4, 128);
    auto kern = k_spmv_ring<MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int grid = (p.n_slices + nw - 1) / nw;
    if (grid > c->n_sm) grid = c->n_sm;
    kern<<<grid, nw * 32, smem, c->stream>>>(p);
    return cudaGetLastError();
  }
  const int per_block = kSpmvThreads / 32;
  int grid = (p.n_slices + per_block - 1) / per_block;
  if (grid > c->spmv_grid) grid = c->spmv_grid;
  if (grid < 1) grid = 1;
  if (c->x_in_smem) {
    const size_t smem = (size_t)c->n_bl * sizeof(float);
    auto kern = k_spmv_sell<true, MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kSpmvThreads, smem, c->stream>>>(p);
  } else {
    k_spmv_sell<false, MODE><<<grid, kSpmvThreads, 0, c->stream>>>(p);
  }
  return cudaGetLastError();
}

cudaError_t launch_spmv(Ctx *c, SpmvMode mode, const float *x, float *out, const int32_t *skip, int32_t a_col) {
  switch (mode) {
    case kSpmvObjective: return launch_spmv_mode<kSpmvObjective>(c, x, out, skip, a_col);
    case kSpmvPlain: return launch_spmv_mode<kSpmvPlain>(c, x, out, skip, a_col);
    case kSpmvColumn: return launch_spmv_mode<kSpmvColumn>(c, x, out, skip, a_col);
    default: return launch_spmv_mode<kSpmvPlainUserOrder>(c, x, out, skip, a_col);
  }
}

// Decide which SpMV variant a context uses: the TMA ring with as many warps as fit beside x.
void spmv_configure(Ctx *c) {
  c->x_in_smem = c->n_bl <= kSpmvXSmemMax;
  c->spmv_grid = c->n_sm * 2;
  c->spmv_ring_warps = 0;
  if (c->opt.reserved & 1) return;                       // test hook: force the direct-load variant
  const size_t budget = 227 * 1024 - 12 * 1024;          // dynamic smem left beside the static tables
  const size_t xbytes = align_up((size_t)c->n_bl * 4, 128);
  for (int nw = kSpmvRingThreads / 32; nw >= 8; nw -= 2) {
    const size_t need = (size_t)nw * kRingStages * kRingStageBytes + align_up((size_t)nw * kRingStages * 8, 128) + xbytes;
    if (need <= budget) { c->spmv_ring_warps = nw; break; }
  }
}

}  // namespace dao
