// dao_master.cu -- step 8, the restricted master problem  min_{y >= 0} F(A y)
// by gradient projection, kept entirely on the device: ONE persistent cooperative kernel, one CTA
// per SM, each CTA owning a fixed slab of voxels.  The slab's dose z, search image dz (fp64) and
// structure ids live in shared memory for the whole solve; the dense aperture-dose block A streams
// through a shared-memory ring filled by a dedicated producer warp with cp.async.bulk (TMA 1-D
// copies, one 16 KB stage per aperture column and tile), so that ~100 KB per SM are in flight
// whatever the register count.  Every pass over A reads the same stage sequence, so the producer
// simply runs ahead: the first stages of the next pass are already resident while the grid
// reduces.  Per projected-gradient iteration:
//   G  z <- z + t dz, g = dF/dz on the slab, grad_k = a_k . g   -> one pass over A, one grid reduction
//   P  every CTA derives the same search direction p (projected steepest descent, optionally
//      with Polak-Ribiere+ conjugation on the free face) from the reduced gradient
//   D  dz = A p on the slab, curvature phi''(0)                  -> one pass over A, one grid reduction
//   L  safeguarded Newton search for the root of phi'(t) = dz . g(z + t dz) on [0, t_max]
//                                                                -> shared memory only
// Grid reductions carry their data in flagged 16-byte slots ({lo32, epoch, hi32, epoch}): a
// reader polls the data itself, there is no counter and no separate release/acquire hop.  Small
// reductions (<= 8 values) are one hop (every CTA reads every CTA's slot); the gradient reduction
// is two hops (CTA i sums value i over the grid in CTA order and publishes it).  All sums are fp64
// in a fixed order: bit-reproducible, identical in every CTA.
// The paper defers the step rule to Men et al. 2009 / Bazaraa et al.; the rule used
// here is DESIGN.md reading S2.
#include "dao_internal.cuh"
#include "dao_ptx.cuh"
#include "dao_grid_reduce.cuh"

#include <math_constants.h>

#include <algorithm>
#include <cstdlib>

namespace dao {

struct MasterParams {
  const float *A;
  int32_t n_vox_pad;
  int32_t slab;            // voxels per CTA (multiple of 128)
  int32_t n_stages;        // ring stages of kMasterStageBytes
  int32_t z_in_smem;       // 1: z, dz, sid of the slab live in shared memory
  int32_t n_struct;
  const uint8_t *sid;
  const float *vt;         // per-voxel thresholds T_j (re-optimisation mode) or null
  const StructEntry *stab;
  double *mz;
  double *mdz;
  double *y;
  uint4 *ll_part;          // [2][grid][kMaxRedux] flagged slots
  uint4 *ll_result;        // [2][kMaxRedux]
  uint32_t *epoch;         // reduction counter, survives dao_reset
  int32_t red_stride;      // slots per CTA in ll_part
  unsigned long long *prof;  // optional [kMasterProfSlots] phase timers (ns), CTA 0 only
  DevState *st;
  dao_iter_record *history;
  const int32_t *ap_beam;
  int32_t add_candidate;
  int32_t max_iter;
  int32_t method;
  int32_t k_max;
  double tol;
  double ls_tol;           // |phi'(t)| <= ls_tol * |phi'(0)| accepts a step
};

// Block-wide sums of NV per-thread doubles -> vals[0..NV) (fixed order: shuffle tree, then warps in order)
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *scratch /*[kNW*NV]*/, double *vals) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const double s = warp_sum_f64(v[i]);
    if (lane == 0) scratch[warp * NV + i] = s;
  }
  wsync();
  if (threadIdx.x < NV) {
    double s = 0.0;
    for (int w = 0; w < kNW; ++w) s += scratch[w * NV + threadIdx.x];
    vals[threadIdx.x] = s;
  }
  wsync();
}

// Transposed butterfly: every lane holds 8 partial sums d[0..8); afterwards every lane of quad q
// (= lane >> 2) holds the warp total of value  (q & 1) + 2 ((q >> 1) & 1) + 4 ((q >> 2) & 1)
// ... i.e. value index bit0 = lane bit 2, bit1 = lane bit 3, bit2 = lane bit 4.  9 shuffles
// instead of 40.
__device__ __forceinline__ double butterfly8(const double (&d)[8], int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  double e[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const double mine = b4 ? d[j + 4] : d[j], other = b4 ? d[j] : d[j + 4];
    e[j] = mine + __shfl_xor_sync(0xffffffffu, other, 16);
  }
  double f[2];
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const double mine = b3 ? e[j + 2] : e[j], other = b3 ? e[j] : e[j + 2];
    f[j] = mine + __shfl_xor_sync(0xffffffffu, other, 8);
  }
  double g = (b2 ? f[1] : f[0]) + __shfl_xor_sync(0xffffffffu, b2 ? f[0] : f[1], 4);
  g += __shfl_xor_sync(0xffffffffu, g, 2);
  g += __shfl_xor_sync(0xffffffffu, g, 1);
  return g;
}
__device__ __forceinline__ int butterfly8_index(int lane) {
  return ((lane >> 2) & 1) | (((lane >> 3) & 1) << 1) | (((lane >> 4) & 1) << 2);
}


// Phase P: the search direction from the reduced gradient (one warp; every CTA computes the same).
// Lane l holds the apertures l, l + 32, ... in registers.  Outputs: p_s (direction, fp32-representable
// values), pgold_s, free_prev_s, and the scalars sc[1] slope phi'(0), sc[2] t_max, sc[3] max|pg|, sc[4] KKT
// residual, si[0] stop, si[1] stopped by the iteration cap, si[2] index of the blocking variable, si[3]
// restarted, si[4] no descent direction left.
__device__ __noinline__ void master_direction(int K, int iters, bool force_restart, int since_restart, int method,
                                              int max_iter, double tol, double F, const double *y_s,
                                              const double *grad_s, double *pgold_s, double *p_s, double *sc, int *si,
                                              unsigned *free_prev_s) {
  const int lane = threadIdx.x & 31;
  const int nq = (K + 31) >> 5;
  double yk[4], gk[4], pgk[4], pk[4], pprev[4];
  double pg_max = 0.0, y_max = 1.0, kkt_l = 0.0, num = 0.0, den = 0.0;
  bool same_free = true;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    yk[q] = 0.0; gk[q] = 0.0; pgk[q] = 0.0; pk[q] = 0.0; pprev[q] = 0.0;
    if (q < nq) {
      const int k = q * 32 + lane;
      bool fr = false;
      if (k < K) {
        gk[q] = grad_s[k]; yk[q] = y_s[k]; pprev[q] = p_s[k];
        const double pold = pgold_s[k];
        fr = (yk[q] > 0.0) || (gk[q] < 0.0);
        pgk[q] = fr ? -gk[q] : 0.0;
        pg_max = fmax(pg_max, fabs(pgk[q]));
        y_max = fmax(y_max, yk[q]);
        kkt_l = fmax(kkt_l, (yk[q] > 0.0) ? fabs(gk[q]) : fmax(-gk[q], 0.0));
        num += pgk[q] * (pgk[q] - pold);
        den += pold * pold;
      }
      const unsigned fn = __ballot_sync(0xffffffffu, fr);
      same_free = same_free && (fn == free_prev_s[q]);
      __syncwarp();
      if (lane == 0) free_prev_s[q] = fn;
    }
  }
  pg_max = warp_max_d(pg_max);
  y_max = warp_max_d(y_max);
  kkt_l = warp_max_d(kkt_l);
  num = warp_sum_f64(num);
  den = warp_sum_f64(den);
  const bool conv = pg_max * y_max <= tol * fmax(F, 1e-300);
  const bool stop = conv || iters >= max_iter;
  bool restart = force_restart || !same_free || method == 0 || since_restart >= K + 8 || !(den > 0.0);
  double beta = 0.0;
  if (!restart) beta = fmax(num / den, 0.0);
  if (beta == 0.0) restart = true;
  // direction, rounded to fp32-representable values
  double slope = 0.0;
  bool infeasible = false;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    double v = pgk[q];
    if (!restart && v != 0.0) v = fma(beta, pprev[q], v);
    v = (double)(float)v;
    if (v < 0.0 && !(yk[q] > 0.0)) infeasible = true;
    slope = fma(v, gk[q], slope);
    pk[q] = v;
  }
  slope = warp_sum_f64(slope);
  infeasible = __any_sync(0xffffffffu, infeasible);
  if (!restart && (infeasible || !(slope < 0.0))) {
    restart = true;
    slope = 0.0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      pk[q] = (double)(float)pgk[q];
      slope = fma(pk[q], gk[q], slope);
    }
    slope = warp_sum_f64(slope);
  }
  double tmax = CUDART_INF;
  int kb = 0x7fffffff;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int k = q * 32 + lane;
    if (k < K) {
      p_s[k] = pk[q];
      pgold_s[k] = pgk[q];
      if (pk[q] < 0.0) {
        const double tk = yk[q] / (-pk[q]);
        if (tk < tmax) { tmax = tk; kb = k; }
      }
    }
  }
  {
    const double tmin = warp_min_d(tmax);
    // smallest k among the lanes that attain the minimum
    int cand_k = (tmax == tmin) ? kb : 0x7fffffff;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cand_k = min(cand_k, __shfl_xor_sync(0xffffffffu, cand_k, o));
    tmax = tmin;
    kb = cand_k;
  }
  if (lane == 0) {
    sc[1] = slope; sc[2] = tmax; sc[3] = pg_max; sc[4] = kkt_l;
    si[0] = stop ? 1 : 0; si[1] = (stop && !conv) ? 1 : 0; si[2] = kb; si[3] = restart ? 1 : 0;
    si[4] = (!(slope < 0.0)) ? 1 : 0;
  }
}

// ---- the A stream ----------------------------------------------------------------------------
// Stage sequence of ONE pass: for tile (kMasterTileVox voxels of the slab) { for k < K { A[k][tile] } }.
// The producer repeats that sequence for ever; consumers walk it with the same counters.
struct MasterSmem {          // carved from dynamic shared memory by every thread identically
  unsigned char *ring;       // [n_stages][kMasterStageBytes]
  uint64_t *full, *empty;    // [n_stages]
  double *zs, *dzs;          // [slab] (shared or this CTA's part of the global arrays)
  const uint8_t *sids;       // [slab]
  const float *vts;          // [slab] or null
  StructEntry *stab;         // [n_struct]
  double *warp_part;         // [kNW][kpad]
};

__global__ void __launch_bounds__(kMasterThreads, kMasterCtasPerSm) k_master(MasterParams p) {
  extern __shared__ __align__(128) unsigned char dyn_smem[];
  // ---- shared state (replicated in every CTA, evolves identically everywhere) ----
  __shared__ double y_s[DAO_MAX_APERTURES];
  __shared__ double grad_s[kMaxRedux];
  __shared__ double pgold_s[DAO_MAX_APERTURES];
  __shared__ double p_s[DAO_MAX_APERTURES];        // search direction (fp32-representable values)
  __shared__ double vals_s[kMaxRedux];
  __shared__ double red_s[kMaxRedux];
  __shared__ double scratch_s[kNW * 4];            // >= kNW * 3
  __shared__ double sc[16];                        // broadcast scalars
  __shared__ int si[8];
  __shared__ unsigned free_prev_s[4];
  __shared__ volatile int s_stop;
  __shared__ volatile unsigned s_consumed_stage, s_consumed_phase;
  __shared__ unsigned long long prof_s[kMasterProfSlots];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int K0 = p.st->K;
  const int cand = p.st->cand_valid;
  const int added = (p.add_candidate && cand) ? 1 : 0;
  const int K = K0 + added;
  if ((p.add_candidate && !added) || K == 0) {     // converged, pool full or empty pool: nothing to do
    if (blockIdx.x == 0 && tid == 0) { p.st->m_added = 0; p.st->m_iters = 0; p.st->m_passes = 0; }
    return;
  }

  // slab of voxels owned by this CTA
  const int vpad = p.n_vox_pad;
  const long long v0l = (long long)blockIdx.x * p.slab;
  const int v0 = (int)(v0l < vpad ? v0l : vpad);
  const int v1 = (v0 + p.slab < vpad) ? v0 + p.slab : vpad;
  const int slab_len = v1 - v0;                                      // multiple of 128 (vpad is)
  const int n_tiles = (slab_len + kMasterTileVox - 1) / kMasterTileVox;
  const int NS = p.n_stages;

  MasterSmem sm;
  {
    unsigned char *q = dyn_smem;
    sm.ring = q; q += (size_t)NS * kMasterStageBytes;
    sm.full = reinterpret_cast<uint64_t *>(q); q += align_up_c((size_t)NS * 8, 128);
    sm.empty = reinterpret_cast<uint64_t *>(q); q += align_up_c((size_t)NS * 8, 128);
    sm.stab = reinterpret_cast<StructEntry *>(q); q += align_up_c((size_t)p.n_struct * sizeof(StructEntry), 128);
    sm.warp_part = reinterpret_cast<double *>(q); q += (size_t)kNW * DAO_MAX_APERTURES * 8;
    if (p.z_in_smem) {
      sm.zs = reinterpret_cast<double *>(q); q += (size_t)p.slab * 8;
      sm.dzs = reinterpret_cast<double *>(q); q += (size_t)p.slab * 8;
      sm.vts = p.vt ? reinterpret_cast<const float *>(q) : nullptr; q += p.vt ? (size_t)p.slab * 4 : 0;
      sm.sids = q;
    } else {
      sm.zs = p.mz + v0; sm.dzs = p.mdz + v0; sm.sids = p.sid + v0;
      sm.vts = p.vt ? p.vt + v0 : nullptr;
    }
  }
  if (tid == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kNW); }
    s_stop = 0;
    for (int i = 0; i < kMasterProfSlots; ++i) prof_s[i] = 0ull;
  }
  fence_mbar_init();
  __syncthreads();

  // =============================== producer warp ================================================
  if (warp == kNW) {
    if (lane == 0) {
      RingPos pp{0, 0u};
      bool first_round = true;
      bool stop = slab_len == 0;
      // Pass i walks the block forwards (tiles and columns ascending) when i is even and backwards when
      // it is odd: what the previous pass read last is read first, so an LRU-like L2 keeps serving the
      // most recent part of A when 4 V K bytes no longer fit it (cyclic order would miss everywhere).
      for (unsigned pass = 0; !stop; ++pass) {
        const bool rev = (pass & 1u) != 0u;
        for (int ti = 0; ti < n_tiles && !stop; ++ti) {
          const int tile = rev ? n_tiles - 1 - ti : ti;
          const int t0 = tile * kMasterTileVox;
          const uint32_t bytes = (uint32_t)min(kMasterTileVox, slab_len - t0) * 4u;
          const float *src = p.A + (size_t)v0 + (size_t)t0;
          for (int kj = 0; kj < K; kj += kMasterColsPerStage) {
            const int ncol = min(kMasterColsPerStage, K - kj);
            if (!first_round) {
              while (!mbar_try_wait(&sm.empty[pp.stage], pp.phase ^ 1u)) {
                if (s_stop) { stop = true; break; }
              }
              if (stop) break;
            }
            mbar_arrive_expect_tx(&sm.full[pp.stage], bytes * (uint32_t)ncol);
            for (int u = 0; u < ncol; ++u) {
              const int k = rev ? K - 1 - (kj + u) : kj + u;
              bulk_g2s(sm.ring + (size_t)pp.stage * kMasterStageBytes + (size_t)u * kMasterColBytes, src + (size_t)k * vpad,
                       bytes, &sm.full[pp.stage]);
            }
            pp.advance(NS);
            if (pp.stage == 0) first_round = false;
          }
        }
      }
      if (slab_len == 0) {
        while (!s_stop) { __nanosleep(200); }
      } else {
        // drain: every issued stage must have landed before the CTA may exit
        while (!s_stop) { __nanosleep(100); }
        RingPos cp{(int)s_consumed_stage, s_consumed_phase};
        while (cp.stage != pp.stage || cp.phase != pp.phase) {
          mbar_wait(&sm.full[cp.stage], cp.phase);
          cp.advance(NS);
        }
      }
    }
    __syncthreads();     // matches the final barrier of the workers
    return;
  }

  // =============================== worker warps =================================================
  for (int i = tid; i < p.n_struct; i += kMasterWorkers) sm.stab[i] = p.stab[i];
  if (tid < DAO_MAX_APERTURES) {
    y_s[tid] = (tid < K0) ? p.y[tid] : 0.0;
    pgold_s[tid] = 0.0;
    p_s[tid] = 0.0;
  }
  if (tid < 4) free_prev_s[tid] = 0u;
  if (p.z_in_smem) {
    uint8_t *sids = const_cast<uint8_t *>(sm.sids);
    float *vts = const_cast<float *>(sm.vts);
    for (int j = tid; j < slab_len; j += kMasterWorkers) {    // j = position, see pos()
      const int i = v0 + (j & ~127) + (j & 31) * 4 + ((j >> 5) & 3);
      sids[j] = p.sid[i];
      if (vts) vts[j] = p.vt[i];
    }
  }
  Reducer red{p.ll_part, p.ll_result, 0u, p.red_stride};
  if (tid == 0) si[7] = (int)*p.epoch;
  wsync();
  red.ep = (uint32_t)si[7];

  const bool prof = (p.prof != nullptr) && blockIdx.x == 0 && tid == 0;
  unsigned long long tprof = prof ? gtimer() : 0ull;
#define PROF_MARK(slot)                                   \
  do {                                                    \
    if (prof) {                                           \
      const unsigned long long now_ = gtimer();           \
      prof_s[slot] += now_ - tprof;                       \
      tprof = now_;                                       \
    }                                                     \
  } while (0)

  RingPos cp{0, 0u};                       // consumer position in the A stream
  unsigned pass_no = 0;                    // passes consumed so far: the parity gives the traversal direction
  // strips of this warp inside a tile: warp and warp + kNW (128 voxels each, 4 per lane)
  const int l0 = warp * 128 + lane * 4, l1 = (warp + kNW) * 128 + lane * 4;

  // Position of voxel (strip, lane, u) of the slab in the z / dz / sid arrays.  In shared memory the 4
  // voxels of a lane are stored 32 doubles apart (conflict-free 64-bit accesses); in global memory
  // (slab too large for shared memory) the order is the plain voxel order.
  const bool permuted = p.z_in_smem != 0;
  auto pos = [&](int strip_base, int u) { return permuted ? strip_base + u * 32 + lane : strip_base + lane * 4 + u; };

  // one D-type pass: out[i] = sum_k coef[k] A[k][i] on the slab (fp64, k in the order of the pass).  With
  // t_commit != 0 the pending step is committed first: z += t_commit * out_old (same thread, same
  // voxels).  With curv, returns this thread's part of phi''(0) = sum 2 c_j out_j^2.
  auto pass_d = [&](const double *coef, double *out, double t_commit, bool curv) -> double {
    double h_acc = 0.0;
    const bool rev = (pass_no++ & 1u) != 0u;
    for (int ti = 0; ti < n_tiles; ++ti) {
      const int tile = rev ? n_tiles - 1 - ti : ti;
      const int t0 = tile * kMasterTileVox;
      const int tn = min(kMasterTileVox, slab_len - t0);
      const bool a0 = l0 < tn, a1 = (kMasterStrips > 1) && l1 < tn;
      double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
      // two stages per step: both waits first, then all loads, then the arithmetic (more independent
      // work per warp between two barrier round trips; four stages per step measured slower: registers)
      for (int k = 0; k < K; k += 2) {
        const bool two = k + 1 < K;
        const double c0 = coef[rev ? K - 1 - k : k], c1 = two ? coef[rev ? K - 2 - k : k + 1] : 0.0;
        const int kin = k % kMasterColsPerStage;           // position of this pair inside its stage
        if (kin == 0) {
          const long long tw = prof ? clock64() : 0ll;
          mbar_wait(&sm.full[cp.stage], cp.phase);
          if (prof) prof_s[13] += (unsigned long long)(clock64() - tw);               // time this thread waited for A in D passes
        }
        const unsigned char *s0 = sm.ring + (size_t)cp.stage * kMasterStageBytes + (size_t)kin * kMasterColBytes;
        const unsigned char *s1 = s0 + kMasterColBytes;
        float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f), x1 = x0, y0 = x0, y1 = x0;
        if (a0) { x0 = *reinterpret_cast<const float4 *>(s0 + (size_t)l0 * 4); if (two) y0 = *reinterpret_cast<const float4 *>(s1 + (size_t)l0 * 4); }
        if (a1) { x1 = *reinterpret_cast<const float4 *>(s0 + (size_t)l1 * 4); if (two) y1 = *reinterpret_cast<const float4 *>(s1 + (size_t)l1 * 4); }
        acc[0] = fma(c0, (double)x0.x, acc[0]); acc[1] = fma(c0, (double)x0.y, acc[1]);
        acc[2] = fma(c0, (double)x0.z, acc[2]); acc[3] = fma(c0, (double)x0.w, acc[3]);
        acc[4] = fma(c0, (double)x1.x, acc[4]); acc[5] = fma(c0, (double)x1.y, acc[5]);
        acc[6] = fma(c0, (double)x1.z, acc[6]); acc[7] = fma(c0, (double)x1.w, acc[7]);
        acc[0] = fma(c1, (double)y0.x, acc[0]); acc[1] = fma(c1, (double)y0.y, acc[1]);
        acc[2] = fma(c1, (double)y0.z, acc[2]); acc[3] = fma(c1, (double)y0.w, acc[3]);
        acc[4] = fma(c1, (double)y1.x, acc[4]); acc[5] = fma(c1, (double)y1.y, acc[5]);
        acc[6] = fma(c1, (double)y1.z, acc[6]); acc[7] = fma(c1, (double)y1.w, acc[7]);
        if (kin == kMasterColsPerStage - 2 || k + 2 >= K) {   // done with the stage
          __syncwarp();
          if (lane == 0) mbar_arrive(&sm.empty[cp.stage]);
          cp.advance(NS);
        }
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (h ? a1 : a0) {
          const int sb = t0 + (h ? warp + kNW : warp) * 128;
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = pos(sb, u);
            const double dd = acc[h * 4 + u];
            if (curv) {
              double z = sm.zs[i];
              if (t_commit != 0.0) { z = fma(t_commit, out[i], z); sm.zs[i] = z; }
              const int s = sm.sids[i];
              if (s != kNoStruct) {
                StructEntry e = sm.stab[s];
              if (sm.vts) e.tm = e.tp = (double)sm.vts[i];
                const double c = (z < e.tm ? e.a : 0.0) + (z > e.tp ? e.b : 0.0);
                h_acc = fma(2.0 * c * dd, dd, h_acc);
              }
            }
            out[i] = dd;
          }
        }
      }
    }
    return h_acc;
  };

  // ---- z = A y on the slab (fp64), dz = 0 ----
  {
    bool any = false;
    for (int k = 0; k < K0; ++k) any = any || (y_s[k] != 0.0);
    if (any) {
      pass_d(y_s, sm.zs, 0.0, false);
    } else {
      for (int i = tid; i < slab_len; i += kMasterWorkers) sm.zs[i] = 0.0;
    }
    for (int i = tid; i < slab_len; i += kMasterWorkers) sm.dzs[i] = 0.0;
  }
  wsync();
  PROF_MARK(0);

  // The step t along the current direction is NOT verified by a separate line-search evaluation:
  // the next gradient pass runs at the trial point z + t dz and delivers phi'(t) = dz . g(z + t dz)
  // (= p . grad) and phi''(t) with the same reduction.  Only when the trial point fails the test
  // |phi'(t)| <= ls_tol |phi'(0)| is t refined (shared memory only) and the pass repeated.
  double t_trial = 0.0;         // step of the trial point (0: no direction yet)
  double slope0 = 0.0, tmax = CUDART_INF;
  int kb = 0x7fffffff;
  bool have_dir = false, forced = false;
  int iters = 0, restarts = 0, since_restart = 0;
  bool force_restart = true;
  int hit_max = 0;
  int passes = (int)pass_no;    // passes over A so far (the initial z = A y, if any)
  double F = CUDART_INF, kkt = 0.0, pgmax = 0.0;

  for (;;) {
    // ============ phase G: g(z + t dz), grad = A^T g, F, phi'(t), phi''(t) ================
    double f_acc = 0.0, s1_acc = 0.0, s2_acc = 0.0;
    ++passes;
    const bool rev = (pass_no++ & 1u) != 0u;
    for (int ti = 0; ti < n_tiles; ++ti) {
      const int tile = rev ? n_tiles - 1 - ti : ti;
      const int t0 = tile * kMasterTileVox;
      const int tn = min(kMasterTileVox, slab_len - t0);
      const bool a0 = l0 < tn, a1 = (kMasterStrips > 1) && l1 < tn;
      double g[8];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const bool act = h ? a1 : a0;
        const int sb = t0 + (h ? warp + kNW : warp) * 128;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          double gv = 0.0;
          if (act) {
            const int i = pos(sb, u);
            const int s = sm.sids[i];
            if (s != kNoStruct) {
              StructEntry e = sm.stab[s];
              if (sm.vts) e.tm = e.tp = (double)sm.vts[i];
              const double dz = sm.dzs[i];
              const double z = fma(t_trial, dz, sm.zs[i]);
              const double un = fmax(e.tm - z, 0.0), ov = fmax(z - e.tp, 0.0);
              f_acc += e.a * un * un + e.b * ov * ov;
              gv = -2.0 * e.a * un + 2.0 * e.b * ov;
              const double c = (un > 0.0 ? e.a : 0.0) + (ov > 0.0 ? e.b : 0.0);
              s1_acc = fma(dz, gv, s1_acc);
              s2_acc = fma(2.0 * c * dz, dz, s2_acc);
            }
          }
          g[h * 4 + u] = gv;
        }
      }
      for (int kb8 = 0; kb8 < K; kb8 += 8) {
        double d[8];
#pragma unroll
        for (int j = 0; j < 8; j += 2) {
          d[j] = 0.0;
          d[j + 1] = 0.0;
          if (kb8 + j < K) {                       // two stages per step: waits, then loads, then arithmetic
            const bool two = kb8 + j + 1 < K;
            const int kin = (kb8 + j) % kMasterColsPerStage;   // position of this pair inside its stage
            if (kin == 0) {
              const long long tw = prof ? clock64() : 0ll;
              mbar_wait(&sm.full[cp.stage], cp.phase);
              if (prof) prof_s[12] += (unsigned long long)(clock64() - tw);           // time this thread waited for A in G passes
            }
            const unsigned char *s0 = sm.ring + (size_t)cp.stage * kMasterStageBytes + (size_t)kin * kMasterColBytes;
            const unsigned char *s1 = s0 + kMasterColBytes;
            float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f), x1 = x0, y0 = x0, y1 = x0;
            if (a0) { x0 = *reinterpret_cast<const float4 *>(s0 + (size_t)l0 * 4); if (two) y0 = *reinterpret_cast<const float4 *>(s1 + (size_t)l0 * 4); }
            if (a1) { x1 = *reinterpret_cast<const float4 *>(s0 + (size_t)l1 * 4); if (two) y1 = *reinterpret_cast<const float4 *>(s1 + (size_t)l1 * 4); }
            {
              double q = (double)x0.x * g[0];
              q = fma((double)x0.y, g[1], q); q = fma((double)x0.z, g[2], q); q = fma((double)x0.w, g[3], q);
              double r = (double)x1.x * g[4];
              r = fma((double)x1.y, g[5], r); r = fma((double)x1.z, g[6], r); r = fma((double)x1.w, g[7], r);
              d[j] = a0 ? (a1 ? q + r : q) : (a1 ? 0.0 + r : 0.0);
            }
            {
              double q = (double)y0.x * g[0];
              q = fma((double)y0.y, g[1], q); q = fma((double)y0.z, g[2], q); q = fma((double)y0.w, g[3], q);
              double r = (double)y1.x * g[4];
              r = fma((double)y1.y, g[5], r); r = fma((double)y1.z, g[6], r); r = fma((double)y1.w, g[7], r);
              d[j + 1] = a0 ? (a1 ? q + r : q) : (a1 ? 0.0 + r : 0.0);
            }
            if (kin == kMasterColsPerStage - 2 || kb8 + j + 2 >= K) {   // done with the stage
              __syncwarp();
              if (lane == 0) mbar_arrive(&sm.empty[cp.stage]);
              cp.advance(NS);
            }
          }
        }
        const double r = butterfly8(d, lane);
        const int kj = kb8 + butterfly8_index(lane);       // position in the pass; column k = kj or K - 1 - kj
        const int kk = rev ? K - 1 - kj : kj;
        if ((lane & 3) == 0 && kj < K) {
          double *slot = sm.warp_part + warp * DAO_MAX_APERTURES + kk;
          *slot = (ti == 0) ? r : (*slot + r);
        }
      }
    }
    {
      const double fs = warp_sum_f64(f_acc), s1 = warp_sum_f64(s1_acc), s2 = warp_sum_f64(s2_acc);
      if (lane == 0) { scratch_s[warp * 3] = fs; scratch_s[warp * 3 + 1] = s1; scratch_s[warp * 3 + 2] = s2; }
    }
    wsync();
    if (tid < K) {
      double s = 0.0;
      if (n_tiles > 0)
        for (int w = 0; w < kNW; ++w) s += sm.warp_part[w * DAO_MAX_APERTURES + tid];
      vals_s[tid] = s;
    } else if (tid < K + 3) {
      double s = 0.0;
      for (int w = 0; w < kNW; ++w) s += scratch_s[w * 3 + (tid - K)];
      vals_s[tid] = s;
    }
    wsync();
    PROF_MARK(1);
    red.large(K + 3, vals_s, grad_s /* K grads, F, phi'(t), phi''(t) */);
    const double F_trial = grad_s[K];
    PROF_MARK(2);

    if (have_dir) {
      const double s1 = grad_s[K + 1], s2 = grad_s[K + 2];
      const bool at_bound = (t_trial >= tmax) && (s1 < 0.0);            // still descending at the bound
      const bool ok = forced || ((fabs(s1) <= p.ls_tol * fabs(slope0) || at_bound) && F_trial <= F + 1e-13 * fabs(F));
      if (!ok) {
        // ---- refine t: root of phi'(t) on [0, tmax]; phi' is non-decreasing, piecewise linear ----
        double lo = 0.0, slo = slope0, hi = CUDART_INF, shi = 0.0;
        double t = t_trial, c1 = s1, c2 = s2;
        for (int ls = 0; ls < 40; ++ls) {
          if (fabs(c1) <= p.ls_tol * fabs(slope0)) break;          // exact enough
          double tn;
          if (c1 < 0.0) {
            if (t >= tmax) break;                                    // descending at the bound
            lo = t; slo = c1;
            tn = (c2 > 0.0) ? t - c1 / c2 : 2.0 * t;
            if (hi < CUDART_INF && !(tn < hi)) tn = lo + (hi - lo) * (-slo) / (shi - slo);
            if (tn > tmax) tn = tmax;
          } else {
            hi = t; shi = c1;
            tn = (c2 > 0.0) ? t - c1 / c2 : 0.5 * (lo + hi);
            if (!(tn > lo)) tn = lo + (hi - lo) * (-slo) / (shi - slo);
          }
          if (!(tn > lo) || !(tn < hi)) tn = 0.5 * (lo + (hi < CUDART_INF ? hi : 2.0 * t));
          if (hi < CUDART_INF && (hi - lo) <= 1e-15 * hi) { t = (c1 < 0.0) ? hi : lo; if (t <= 0.0) t = hi; break; }
          if (tn == t) break;
          t = tn;
          double acc2[2] = {0.0, 0.0};   // phi'(t), phi''(t)
          for (int i = tid; i < slab_len; i += kMasterWorkers) {
            const int s = sm.sids[i];
            if (s == kNoStruct) continue;
            StructEntry e = sm.stab[s];
              if (sm.vts) e.tm = e.tp = (double)sm.vts[i];
            const double dz = sm.dzs[i];
            const double z = fma(t, dz, sm.zs[i]);
            const double u = fmax(e.tm - z, 0.0), o = fmax(z - e.tp, 0.0);
            const double gv = -2.0 * e.a * u + 2.0 * e.b * o;
            const double c = (u > 0.0 ? e.a : 0.0) + (o > 0.0 ? e.b : 0.0);
            acc2[0] = fma(dz, gv, acc2[0]);
            acc2[1] = fma(2.0 * c * dz, dz, acc2[1]);
          }
          block_sum<2>(acc2, scratch_s, vals_s);
          red.small(2, vals_s, red_s);
          if (prof) ++prof_s[7];
          c1 = red_s[0]; c2 = red_s[1];
        }
        if (prof) ++prof_s[11];
        t_trial = t;
        forced = true;
        wsync();
        PROF_MARK(6);
        continue;                        // gradient pass again, at the refined step
      }
      // ---- accept: y += t p (every CTA identically); z is committed by the next D pass ----
      if (tid < K) {
        double yk = fma(t_trial, p_s[tid], y_s[tid]);
        if (yk < 0.0) yk = 0.0;
        if (at_bound && tid == kb) yk = 0.0;
        y_s[tid] = yk;
      }
      if (at_bound) force_restart = true;
      ++iters;
      wsync();
    }
    PROF_MARK(14);                       // accept / refine decision and the y update
    F = F_trial;

    // ================= phase P: direction (warp 0, identical in every CTA) ================
    if (warp == 0)
      master_direction(K, iters, force_restart, since_restart, p.method, p.max_iter, p.tol, F, y_s, grad_s, pgold_s,
                       p_s, sc, si, free_prev_s);
    wsync();
    pgmax = sc[3];
    kkt = sc[4];
    PROF_MARK(3);
    if (si[0] || si[4]) {               // converged, iteration cap, or no descent left
      hit_max = si[1];
      if (t_trial != 0.0) {             // commit the accepted step
        for (int i = tid; i < slab_len; i += kMasterWorkers) sm.zs[i] = fma(t_trial, sm.dzs[i], sm.zs[i]);
      }
      break;
    }
    slope0 = sc[1]; tmax = sc[2];
    kb = si[2];
    if (si[3]) { ++restarts; since_restart = 0; } else { ++since_restart; }
    force_restart = false;

    // ================= phase D: commit z, dz = A p, curvature =============================
    ++passes;
    const double h_acc = pass_d(p_s, sm.dzs, t_trial, true);
    {
      double hv[1] = {h_acc};
      block_sum<1>(hv, scratch_s, vals_s);
    }
    PROF_MARK(4);
    red.small(1, vals_s, red_s);
    const double h0 = red_s[0];
    PROF_MARK(5);
    // Newton step on the ray (exact while the voxel active set does not change), clipped to the bound
    double t = (h0 > 0.0) ? (-slope0 / h0) : ((tmax < CUDART_INF) ? tmax : 1.0);
    if (t > tmax) t = tmax;
    t_trial = t;
    have_dir = true;
    forced = false;
  }
  wsync();

  // ---- publish ----
  if (p.z_in_smem) {
    for (int j = tid; j < slab_len; j += kMasterWorkers) {
      const int i = (j & ~127) + (j & 31) * 4 + ((j >> 5) & 3);
      p.mz[v0 + i] = sm.zs[j];
      p.mdz[v0 + i] = sm.dzs[j];
    }
  }
  if (tid == 0) {
    s_consumed_stage = (unsigned)cp.stage;
    s_consumed_phase = cp.phase;
    __threadfence_block();
    s_stop = 1;
  }
  if (blockIdx.x == 0) {
    if (tid < K) p.y[tid] = y_s[tid];
    if (tid == 0) {
      *p.epoch = red.ep;
      if (p.prof) {
        prof_s[8] += (unsigned long long)iters;
        prof_s[9] += 1ull;
        PROF_MARK(10);
        for (int i = 0; i < kMasterProfSlots; ++i) p.prof[i] += prof_s[i];
      }
      DevState *st = p.st;
      st->K = K;
      st->m_iters = iters;
      st->m_passes = passes;             // gradient passes (incl. repeated ones after a refined step) + dz passes
      st->pass_total += passes;
      st->m_hit_max = hit_max;
      st->n_hit_max += hit_max ? 1 : 0;
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
        rec.n_passes = passes;
        rec.hit_max_iter = hit_max;
        p.history[K - 1] = rec;
      }
    }
  }
#undef PROF_MARK
  __syncthreads();       // the producer warp joins after draining the ring
}

// Shared-memory plan: static tables + ring + (when it fits) the slab's z, dz, sid.
static size_t master_fixed_smem(const Ctx *c, int n_stages) {
  return (size_t)n_stages * kMasterStageBytes + 2 * align_up((size_t)n_stages * 8, 128) +
         align_up((size_t)std::max(c->n_struct, 1) * sizeof(StructEntry), 128) + (size_t)kNW * DAO_MAX_APERTURES * 8;
}

cudaError_t master_configure(Ctx *c) {
  if (c->opt.master_method >= 2) return newton_configure(c);
  c->master_grid = std::min(c->n_sm * kMasterCtasPerSm, kMasterMaxGrid);
  int slab = (c->n_vox_pad + c->master_grid - 1) / c->master_grid;
  slab = (slab + 127) / 128 * 128;
  c->master_slab = slab;
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, k_master);
  if (e != cudaSuccess) return e;
  int max_optin = 0;
  e = cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device);
  if (e != cudaSuccess) return e;
  // shared memory per CTA: the opt-in maximum for one CTA per SM; with more, an equal share of the SM's
  // 228 KB (1 KB per resident CTA is reserved by the system)
  size_t budget = (size_t)max_optin - fa.sharedSizeBytes - 1024;
  if (kMasterCtasPerSm > 1) budget = (size_t)(228 * 1024) / kMasterCtasPerSm - 1024 - fa.sharedSizeBytes - 512;
  const size_t slab_bytes = (size_t)slab * (c->has_vt ? 21 : 17);
  // prefer z in shared memory with >= 4 stages; otherwise z stays in global memory (L2)
  c->master_z_in_smem = 0;
  int stages = 0;
  if (master_fixed_smem(c, 2) + slab_bytes <= budget) {
    c->master_z_in_smem = 1;
    stages = 2;
    while (stages < kMasterMaxStages && master_fixed_smem(c, stages + 1) + slab_bytes <= budget) ++stages;
  } else {
    stages = 2;
    while (stages < kMasterMaxStages && master_fixed_smem(c, stages + 1) <= budget) ++stages;
    if (master_fixed_smem(c, stages) > budget) return cudaErrorLaunchOutOfResources;
  }
  c->master_stages = stages;
  c->master_smem = master_fixed_smem(c, stages) + (c->master_z_in_smem ? align_up(slab_bytes, 128) : 0);
  e = cudaFuncSetAttribute(k_master, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->master_smem);
  if (e != cudaSuccess) return e;
  int nb = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_master, kMasterThreads, c->master_smem);
  if (e != cudaSuccess) return e;
  if (nb < kMasterCtasPerSm) return cudaErrorLaunchOutOfResources;
  return cudaSuccess;
}

cudaError_t launch_master(Ctx *c, bool add_candidate) {
  if (c->opt.master_method >= 2) return launch_newton(c, add_candidate);
  c->x_current = false;                    // methods 0 / 1 leave step 1 (beamlet intensities) to k_intensity
  MasterParams p{};
  p.A = c->d.A;
  p.n_vox_pad = c->n_vox_pad;
  p.slab = c->master_slab;
  p.n_stages = c->master_stages;
  p.z_in_smem = c->master_z_in_smem;
  p.n_struct = std::max(c->n_struct, 1);
  p.sid = c->d.sid;
  p.vt = c->has_vt ? c->d.vt : nullptr;
  p.stab = c->d.stab;
  p.mz = c->d.mz;
  p.mdz = c->d.mdz;
  p.y = c->d.y;
  p.ll_part = c->d.ll_part;
  p.ll_result = c->d.ll_result;
  p.epoch = c->d.m_epoch;
  p.red_stride = c->red_stride;
  p.prof = (c->opt.reserved & 2) ? c->d.m_prof : nullptr;
  p.st = c->d.state;
  p.history = c->d.history;
  p.ap_beam = c->d.ap_beam;
  p.add_candidate = add_candidate ? 1 : 0;
  p.max_iter = c->opt.master_max_iter;
  p.method = c->opt.master_method;
  p.k_max = c->opt.k_max;
  p.tol = c->opt.master_tol;
  p.ls_tol = c->opt.master_ls_tol;
  void *args[] = {&p};
  ++c->n_launches;
  return cudaLaunchCooperativeKernel((void *)k_master, dim3(c->master_grid), dim3(kMasterThreads), args,
                                     c->master_smem, c->stream);
}

}  // namespace dao
