// dao_newton.cu -- step 8 with master_method = 2: the restricted master problem  min_{y >= 0} F(A y)
// by PROJECTED NEWTON on the free variables.  F is a convex piecewise quadratic
// (eq. 3-5, 9-10), so on a fixed voxel active set its Hessian  H = A^T diag(2 c) A,
// c_j = a_j [z_j < T_j^-] + b_j [z_j > T_j^+],  is exact and a Newton step lands on the minimiser of the
// current piece: 4-5 passes over the dose block A per solve instead of ~120 for gradient projection.
// The paper defers the method of the master to Men et al. 2009 / Bazaraa et al.; the RESULT
// (the optimal value) is unique by convexity, and the stopping test is the one of methods 0/1 and of the
// oracle (reading S2), so parity is unaffected by the choice of method.
//
// ONE persistent cooperative kernel, one CTA per SM (16 worker warps + 1 producer warp).  The dose
// block is stored tiled (NewtonLayout): the K live columns of a tile of T voxels are one contiguous
// range, fetched by ONE cp.async.bulk (1-D TMA) into a stage of a shared-memory ring.  With all K
// columns of a tile resident, one pass computes EVERYTHING at a trial point y:
//   Z  z_j = sum_k y_k A[k][j]                        (fp64, thread per voxel and k-slice)
//   P  F, pi_j = dF/dz_j, s_j = 2 c_j, list of the active voxels (s_j != 0) of the tile
//   H  the augmented Gram matrix  [A; pi/s]-style:  H[k1][k2] += sum_j A[k1][j] s_j A[k2][j]  and
//      grad[k1] += sum_j A[k1][j] pi_j  as one extra column, over the ACTIVE voxels only, on the fp64
//      tensor cores (mma.sync m8n8k4 f64: 8x8 blocks of H, 4 voxels per instruction; every warp owns a
//      fixed set of blocks whose accumulators stay in registers for the whole pass)
// then one grid reduction of (H, grad, F) through flagged slots (dao_grid_reduce.cuh), and every CTA
// computes the same Newton step on the free set {k : y_k > 0 or grad_k < 0} by an LDL^T factorisation
// in shared memory.  The trial point y + t d (t = 1 unless a bound is hit first) is accepted on
// sufficient decrease of F -- the next pass IS the evaluation -- else t is shortened by the secant
// of phi'(t) = d . grad(y + t d).  All sums fp64 in a fixed order: bit-reproducible.
#include "dao_internal.cuh"
#include "dao_ptx.cuh"
#include "dao_grid_reduce.cuh"

#include <math_constants.h>

#include <algorithm>

namespace dao {

constexpr int kNwtMaxB = 10;            // 8x8 blocks of H a warp may own (153 blocks at K = 128 over 16 warps)
constexpr int kNwtMaxBlocks = 160;      // >= nb (nb + 1) / 2 for nb = 17
constexpr int kNwtZThreads = kMasterWorkers;

struct NewtonParams {
  const float *A;            // tiled dose block
  int32_t n_vox_pad;
  int32_t T, TP;             // tile voxels, column pitch (floats)
  int64_t tile_stride;       // floats between tiles
  int32_t n_tiles;
  int32_t n_stages;
  int32_t stage_bytes;
  int32_t n_red_cap;         // capacity (doubles) of the reduction staging array = slots per CTA
  int32_t lbuf_doubles;      // capacity of the factorisation buffer
  int32_t n_struct;
  const uint8_t *sid;
  const float *vt;           // per-voxel thresholds T_j (re-optimisation mode) or null
  const StructEntry *stab;
  double *mz;                // [n_vox_pad] z = A y of the last pass (internal order)
  double *y;
  uint4 *ll_part;
  uint4 *ll_result;
  uint32_t *epoch;
  unsigned long long *prof;  // optional phase timers (ns), CTA 0 only
  DevState *st;
  dao_iter_record *history;
  const int32_t *ap_beam;
  int32_t add_candidate;
  int32_t max_iter;
  int32_t k_max;
  double tol;
};

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// index of block (I, J), I <= J < nb, in the row-major enumeration of the upper block triangle
__host__ __device__ __forceinline__ int blk_index(int nb, int I, int J) { return I * nb - (I * (I - 1)) / 2 + (J - I); }

// entry (k1, k2), k1 <= k2, of the reduced augmented matrix
__device__ __forceinline__ double h_at(const double *hred, int nb, int k1, int k2) {
  return hred[blk_index(nb, k1 >> 3, k2 >> 3) * 64 + (k1 & 7) * 8 + (k2 & 7)];
}
__device__ __forceinline__ double h_sym(const double *hred, int nb, int a, int b) {
  return a <= b ? h_at(hred, nb, a, b) : h_at(hred, nb, b, a);
}
// packed lower triangle
__device__ __forceinline__ int lidx(int i, int j) { return (i * (i + 1)) / 2 + j; }

__global__ void __launch_bounds__(kMasterThreads, 1) k_master_newton(NewtonParams p) {
  extern __shared__ __align__(128) unsigned char dyn_smem[];
  __shared__ double y_s[DAO_MAX_APERTURES];        // accepted point
  __shared__ double ytr_s[DAO_MAX_APERTURES];      // trial point of the current pass
  __shared__ double d_s[DAO_MAX_APERTURES];        // Newton direction
  __shared__ double grad_s[DAO_MAX_APERTURES];     // gradient at the accepted point
  __shared__ double dpiv_s[DAO_MAX_APERTURES + 1]; // pivots of the LDL^T factorisation
  __shared__ double xs_s[DAO_MAX_APERTURES + 1];   // solution on the free set
  __shared__ int fr_s[DAO_MAX_APERTURES];          // free variables
  __shared__ unsigned short blk_s[kNwtMaxBlocks];  // block -> (I << 8) | J
  __shared__ double sc[16];
  __shared__ int si[16];
  __shared__ int wcnt_s[kNW];
  __shared__ double fred_s[kNW];
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

  // tiles owned by this CTA: b, b + grid, b + 2 grid, ...  The internal voxel order is sorted by the length of
  // the voxel's row of D, which puts the high-dose (= penalised, "active") voxels first: interleaving gives
  // every CTA the same mix (contiguous ranges were measured 4x slower: the first CTAs did all the H work)
  const int T = p.T, TP = p.TP;
  const int tb0 = (int)blockIdx.x, tstep = (int)gridDim.x;
  const int ntl = (p.n_tiles > tb0) ? (p.n_tiles - tb0 + tstep - 1) / tstep : 0;
  const int NS = p.n_stages;

  // dynamic shared memory
  unsigned char *q = dyn_smem;
  unsigned char *ring = q; q += (size_t)NS * p.stage_bytes;
  uint64_t *full = reinterpret_cast<uint64_t *>(q); q += 128;
  uint64_t *empty = reinterpret_cast<uint64_t *>(q); q += 128;
  StructEntry *stab = reinterpret_cast<StructEntry *>(q); q += align_up_c((size_t)p.n_struct * sizeof(StructEntry), 128);
  double *hred = reinterpret_cast<double *>(q); q += align_up_c((size_t)p.n_red_cap * 8, 128);
  double *lbuf = reinterpret_cast<double *>(q); q += align_up_c((size_t)p.lbuf_doubles * 8, 128);
  double *zpart = reinterpret_cast<double *>(q); q += (size_t)kNwtZThreads * 8;
  double *gs = reinterpret_cast<double *>(q); q += align_up_c((size_t)(T + 4) * 8, 128);
  double *ss = reinterpret_cast<double *>(q); q += align_up_c((size_t)(T + 4) * 8, 128);
  unsigned short *list = reinterpret_cast<unsigned short *>(q);

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kNW); }
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
      bool stop = ntl == 0;
      const uint32_t bytes = (uint32_t)K * (uint32_t)TP * 4u;
      // every pass reads the same tiles; odd passes walk them backwards (what was read last is read
      // first: an LRU-like L2 keeps serving the most recent part of A once 4 V K bytes exceed it)
      for (unsigned pass = 0; !stop; ++pass) {
        const bool rev = (pass & 1u) != 0u;
        for (int ti = 0; ti < ntl && !stop; ++ti) {
          const int tile = tb0 + (rev ? ntl - 1 - ti : ti) * tstep;
          if (!first_round) {
            while (!mbar_try_wait(&empty[pp.stage], pp.phase ^ 1u)) {
              if (s_stop) { stop = true; break; }
            }
            if (stop) break;
          }
          mbar_arrive_expect_tx(&full[pp.stage], bytes);
          bulk_g2s(ring + (size_t)pp.stage * p.stage_bytes, p.A + (size_t)tile * (size_t)p.tile_stride, bytes,
                   &full[pp.stage]);
          pp.advance(NS);
          if (pp.stage == 0) first_round = false;
        }
      }
      while (!s_stop) { __nanosleep(100); }
      if (ntl > 0) {
        // drain: every issued stage must have landed before the CTA may exit
        RingPos cp{(int)s_consumed_stage, s_consumed_phase};
        while (cp.stage != pp.stage || cp.phase != pp.phase) {
          mbar_wait(&full[cp.stage], cp.phase);
          cp.advance(NS);
        }
      }
    }
    __syncthreads();     // matches the final barrier of the workers
    return;
  }

  // =============================== worker warps =================================================
  const int nb = (K + 1 + 7) >> 3;                 // 8x8 block rows of the augmented matrix (K columns + gradient)
  const int nblocks = nb * (nb + 1) / 2;
  const int n_red = nblocks * 64 + 1;              // + F
  for (int i = tid; i < p.n_struct; i += kMasterWorkers) stab[i] = p.stab[i];
  if (tid < DAO_MAX_APERTURES) {
    y_s[tid] = (tid < K0) ? p.y[tid] : 0.0;
    ytr_s[tid] = y_s[tid];
    d_s[tid] = 0.0;
    grad_s[tid] = 0.0;
  }
  for (int bi = tid; bi < nblocks; bi += kMasterWorkers) {   // block table (row-major upper triangle)
    int I = 0, rem = bi;
    while (rem >= nb - I) { rem -= nb - I; ++I; }
    blk_s[bi] = (unsigned short)((I << 8) | (I + rem));
  }
  if (tid < 4) { gs[T + tid] = 0.0; ss[T + tid] = 0.0; }      // the dummy voxel that pads a quad
  Reducer red{p.ll_part, p.ll_result, 0u, p.n_red_cap};
  if (tid == 0) si[7] = (int)*p.epoch;
  wsync();
  red.ep = (uint32_t)si[7];

  // distribution of the H blocks: NC classes of warps x NG groups; class c owns the blocks c, c + NC, ...;
  // group g takes the quads g, g + NG, ... of the active voxels of a tile
  int NC = 1;
  while ((nblocks + NC - 1) / NC > kNwtMaxB || (NC < kNW && (nblocks + NC - 1) / NC > 7 && nblocks >= 2 * NC)) NC <<= 1;
  if (NC > kNW) NC = kNW;
  const int NG = kNW / NC;
  const int cls = warp % NC, grp = warp / NC;
  const int nmine = (nblocks - cls + NC - 1) / NC;     // blocks of this warp
  // Z phase: thread = (k-slice, voxel)
  const int KS = kNwtZThreads / T;                     // k-slices
  const int zs = tid / T, zv = tid - zs * T;
  const int kchunk = (K + KS - 1) / KS;
  const int zk0 = min(K, zs * kchunk), zk1 = min(K, zk0 + kchunk);
  const bool z_on = zs < KS;
  const int fin_warps = T >> 5;                        // warps that finalise voxels (T <= 256)

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

  RingPos cp{0, 0u};
  unsigned pass_no = 0;
  const int rowoff = (lane >> 2) * TP;
  const int r8 = lane >> 2, c2 = (lane & 3) * 2;

  // ---- one pass over A at the point yv: z, F, pi, grad, H -> hred (reduced over the grid) ----
  auto pass = [&](const double *yv) {
    double acc[kNwtMaxB][2];
#pragma unroll
    for (int j = 0; j < kNwtMaxB; ++j) { acc[j][0] = 0.0; acc[j][1] = 0.0; }
    unsigned blk[kNwtMaxB];
#pragma unroll
    for (int j = 0; j < kNwtMaxB; ++j) blk[j] = (j < nmine) ? (unsigned)blk_s[cls + j * NC] : 0u;
    double f_acc = 0.0;
    const bool rev = (pass_no++ & 1u) != 0u;
    for (int ti = 0; ti < ntl; ++ti) {
      const int tile = tb0 + (rev ? ntl - 1 - ti : ti) * tstep;
      mbar_wait(&full[cp.stage], cp.phase);
      const float *M = reinterpret_cast<const float *>(ring + (size_t)cp.stage * p.stage_bytes);
      // ---- Z: partial doses ----
      if (z_on) {
        double a0 = 0.0, a1 = 0.0;
        const float *col = M + zv;
        int k = zk0;
        for (; k + 1 < zk1; k += 2) {
          a0 = fma(yv[k], (double)col[(size_t)k * TP], a0);
          a1 = fma(yv[k + 1], (double)col[(size_t)(k + 1) * TP], a1);
        }
        if (k < zk1) a0 = fma(yv[k], (double)col[(size_t)k * TP], a0);
        zpart[tid] = a0 + a1;
      }
      wsync();
      // ---- P: dose, penalty, gradient, curvature weight, active flag ----
      bool active = false;
      if (tid < T) {
        double z = 0.0;
        for (int s = 0; s < KS; ++s) z += zpart[s * T + tid];
        const int vg = tile * T + tid;
        double gv = 0.0, sv = 0.0;
        if (vg < p.n_vox_pad) {
          const int s = p.sid[vg];
          if (s != kNoStruct) {
            StructEntry e = stab[s];
            if (p.vt) e.tm = e.tp = (double)p.vt[vg];
            const double un = fmax(e.tm - z, 0.0), ov = fmax(z - e.tp, 0.0);
            f_acc += e.a * un * un + e.b * ov * ov;
            gv = -2.0 * e.a * un + 2.0 * e.b * ov;
            sv = 2.0 * ((un > 0.0 ? e.a : 0.0) + (ov > 0.0 ? e.b : 0.0));
          }
          p.mz[vg] = z;
        }
        gs[tid] = gv;
        ss[tid] = sv;
        active = sv != 0.0;
      }
      int rank = 0;
      if (warp < fin_warps) {
        const unsigned m = __ballot_sync(0xffffffffu, active);
        rank = __popc(m & ((1u << lane) - 1u));
        if (lane == 0) wcnt_s[warp] = __popc(m);
      }
      wsync();
      int n_act = 0, my_off = 0;
      for (int w = 0; w < fin_warps; ++w) {
        const int cnt = wcnt_s[w];
        if (w < warp) my_off += cnt;
        n_act += cnt;
      }
      if (active) list[my_off + rank] = (unsigned short)tid;
      if (tid < 4 && n_act + tid < ((n_act + 3) & ~3)) list[n_act + tid] = (unsigned short)T;
      wsync();
      // ---- H: augmented Gram matrix over the active voxels, fp64 tensor cores ----
      const int nq = (n_act + 3) >> 2;
      for (int qd = grp; qd < nq; qd += NG) {
        const int vox = (int)list[qd * 4 + (lane & 3)];
        const double sv = ss[vox], gv = gs[vox];
        const float *Mv = M + rowoff + vox;
#pragma unroll
        for (int j = 0; j < kNwtMaxB; ++j) {
          if (j < nmine) {
            const int I = (int)(blk[j] >> 8), J = (int)(blk[j] & 255u);
            const int ka = I * 8 + r8, kb = J * 8 + r8;
            double a = 0.0, b = 0.0;
            if (ka < K) a = (double)Mv[(size_t)I * 8 * TP];
            if (kb < K) b = sv * (double)Mv[(size_t)J * 8 * TP];
            else if (kb == K) b = gv;
            dmma884(acc[j][0], acc[j][1], a, b);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[cp.stage]);
      cp.advance(NS);
    }
    PROF_MARK(1);
    // ---- CTA partial: the groups add their blocks in group order ----
    for (int gg = 0; gg < NG; ++gg) {
      if (grp == gg) {
#pragma unroll
        for (int j = 0; j < kNwtMaxB; ++j) {
          if (j < nmine) {
            double *h = hred + (size_t)(cls + j * NC) * 64 + r8 * 8 + c2;
            if (gg == 0) { h[0] = acc[j][0]; h[1] = acc[j][1]; }
            else { h[0] += acc[j][0]; h[1] += acc[j][1]; }
          }
        }
      }
      wsync();
    }
    {
      const double fs = warp_sum_f64(f_acc);
      if (lane == 0) fred_s[warp] = fs;
    }
    wsync();
    if (tid == 0) {
      double s = 0.0;
      for (int w = 0; w < kNW; ++w) s += fred_s[w];
      hred[nblocks * 64] = s;
    }
    wsync();
    red.large(n_red, hred, hred);
    PROF_MARK(2);
  };

  // ---- first pass: everything at the warm start (previous optimum, new column at 0) ----
  pass(y_s);
  int passes = 1, iters = 0, hit_max = 0, nbt = 0, stall = 0;
  bool have_dir = false;
  double F = hred[nblocks * 64], t_step = 0.0, slope0 = 0.0, kkt = 0.0, pgmax = 0.0;

  for (;;) {
    // ================= decision on the pass just made (warp 0; identical in every CTA) =================
    if (warp == 0) {
      const double F_t = hred[nblocks * 64];
      int verdict = 1;                                     // 1 accept (or first pass), 0 shorten the step, 2 give up
      if (have_dir) {
        double s1 = 0.0;
        for (int k = lane; k < K; k += 32) s1 = fma(d_s[k], h_at(hred, nb, k, K), s1);
        s1 = warp_sum_f64(s1);
        const bool ok = F_t <= F + 1e-4 * t_step * slope0 + 1e-14 * fabs(F);
        if (!ok) {
          if (nbt >= 40) {
            verdict = 2;
          } else {
            verdict = 0;
            // phi' is non-decreasing and piecewise linear on the segment: secant through phi'(0), phi'(t)
            double tn = (s1 > slope0) ? t_step * (-slope0) / (s1 - slope0) : 0.5 * t_step;
            tn = fmin(fmax(tn, 0.1 * t_step), 0.9 * t_step);
            for (int k = lane; k < K; k += 32) ytr_s[k] = fmax(fma(tn, d_s[k], y_s[k]), 0.0);
            if (lane == 0) sc[0] = tn;
          }
        }
      }
      if (lane == 0) si[0] = verdict;
    }
    wsync();
    PROF_MARK(3);
    const int verdict = si[0];
    if (verdict == 0) {                                    // same direction, shorter step
      t_step = sc[0];
      ++nbt;
      pass(ytr_s);
      ++passes;
      continue;
    }
    if (verdict == 2) {                                    // no acceptable step: restore z = A y and stop
      hit_max = 1;
      pass(y_s);
      ++passes;
      have_dir = false;
    }
    if (have_dir) {
      const double F_t = hred[nblocks * 64];
      stall = (F_t < F - 1e-15 * fabs(F)) ? 0 : stall + 1;
      F = F_t;
      ++iters;
      if (tid < K) y_s[tid] = ytr_s[tid];
    }
    // ================= free set, stopping test =================
    if (warp == 0) {
      double pg_max = 0.0, y_max = 1.0, kkt_l = 0.0;
      int nf = 0;
      for (int k0 = 0; k0 < K; k0 += 32) {
        const int k = k0 + lane;
        bool fr = false;
        if (k < K) {
          const double g = h_at(hred, nb, k, K), yk = have_dir ? ytr_s[k] : y_s[k];
          grad_s[k] = g;
          fr = !(yk <= 0.0 && g >= 0.0);
          pg_max = fmax(pg_max, fr ? fabs(g) : 0.0);
          y_max = fmax(y_max, yk);
          kkt_l = fmax(kkt_l, (yk > 0.0) ? fabs(g) : fmax(-g, 0.0));
        }
        const unsigned m = __ballot_sync(0xffffffffu, fr);
        if (fr) fr_s[nf + __popc(m & ((1u << lane) - 1u))] = k;
        nf += __popc(m);
      }
      pg_max = warp_max_d(pg_max);
      y_max = warp_max_d(y_max);
      kkt_l = warp_max_d(kkt_l);
      const bool conv = pg_max * y_max <= p.tol * fmax(F, 1e-300);
      if (lane == 0) {
        sc[3] = pg_max; sc[4] = kkt_l;
        si[1] = conv ? 1 : 0;
        si[2] = nf;
      }
    }
    wsync();
    pgmax = sc[3];
    kkt = sc[4];
    if (si[1]) break;
    if (hit_max) break;
    if (iters >= p.max_iter || stall >= 3) { hit_max = 1; break; }
    int nf = si[2];

    // ================= Newton direction on the free set: (H_ff + ridge I) x = -grad_f =================
    // LDL^T in the packed lower triangle of lbuf with the right-hand side as an extra row (its entries
    // come out forward-substituted).  A free variable sitting at 0 whose component is negative cannot
    // move: it leaves the free set and the system is solved again.
    bool newton_ok = false;
    for (int round = 0; round < DAO_MAX_APERTURES && nf > 0; ++round) {
      // ridge from the mean diagonal
      if (warp == 0) {
        double tr = 0.0;
        for (int qf = lane; qf < nf; qf += 32) tr += h_at(hred, nb, fr_s[qf], fr_s[qf]);
        tr = warp_sum_f64(tr);
        if (lane == 0) sc[5] = 1e-12 * (tr / nf) + 1e-300;
      }
      wsync();
      const double ridge = sc[5];
      for (int i = warp; i <= nf; i += kNW) {
        for (int j = lane; j <= i && j < nf; j += 32) {
          double v;
          if (i < nf) v = h_sym(hred, nb, fr_s[i], fr_s[j]) + (i == j ? ridge : 0.0);
          else v = -grad_s[fr_s[j]];
          lbuf[lidx(i, j)] = v;
        }
      }
      wsync();
      for (int j = 0; j < nf; ++j) {
        double dj = lbuf[lidx(j, j)];
        if (!(dj > ridge)) dj = ridge;
        if (tid == 0) dpiv_s[j] = dj;
        const double inv = 1.0 / dj;
        // trailing update: rows i in (j, nf], columns k in (j, min(i, nf - 1)]
        const int nrow = nf - j;                           // rows j+1 .. nf
        for (int e = tid; e < nrow * nrow; e += kMasterWorkers) {
          const int i = j + 1 + e / nrow, k = j + 1 + e % nrow;
          if (k <= i && k < nf) lbuf[lidx(i, k)] = fma(-lbuf[lidx(i, j)] * inv, lbuf[lidx(k, j)], lbuf[lidx(i, k)]);
        }
        wsync();
      }
      // back substitution (warp 0): x_i = (u_i - sum_{k > i} c_ki x_k) / d_i, column oriented
      if (warp == 0) {
        double u[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const int i = lane + 32 * m;
          u[m] = (i < nf) ? lbuf[lidx(nf, i)] : 0.0;
        }
        for (int k = nf - 1; k >= 0; --k) {
          const double uk = __shfl_sync(0xffffffffu, (k >> 5) == 0 ? u[0] : (k >> 5) == 1 ? u[1] : (k >> 5) == 2 ? u[2] : u[3], k & 31);
          const double xk = uk / dpiv_s[k];
          if (lane == 0) xs_s[k] = xk;
#pragma unroll
          for (int m = 0; m < 4; ++m) {
            const int i = lane + 32 * m;
            if (i < k) u[m] = fma(-lbuf[lidx(k, i)], xk, u[m]);
          }
        }
        __syncwarp();
        // shrink the free set where a variable at its bound would move out of the feasible set
        int nkeep = 0;
        bool any_drop = false;
        for (int q0 = 0; q0 < nf; q0 += 32) {
          const int qf = q0 + lane;
          bool keep = false;
          int kf = 0;
          double xv = 0.0;
          if (qf < nf) {
            kf = fr_s[qf];
            xv = xs_s[qf];
            keep = !(y_s[kf] <= 0.0 && xv < 0.0);
          }
          const unsigned m = __ballot_sync(0xffffffffu, keep);
          any_drop = any_drop || (__popc(m) != min(32, nf - q0));
          __syncwarp();
          if (keep) { fr_s[nkeep + __popc(m & ((1u << lane) - 1u))] = kf; }
          nkeep += __popc(m);
          __syncwarp();
        }
        if (lane == 0) { si[3] = any_drop ? 1 : 0; si[2] = nkeep; }
      }
      wsync();
      if (!si[3]) { newton_ok = true; break; }
      nf = si[2];
    }
    // ================= direction, step bound, trial point (warp 0) =================
    if (warp == 0) {
      for (int k = lane; k < K; k += 32) d_s[k] = 0.0;
      __syncwarp();
      double slope = 0.0;
      if (newton_ok) {
        for (int qf = lane; qf < nf; qf += 32) {
          const int k = fr_s[qf];
          const double v = xs_s[qf];
          d_s[k] = v;
          slope = fma(v, grad_s[k], slope);
        }
      }
      slope = warp_sum_f64(slope);
      __syncwarp();
      if (!(newton_ok && slope < 0.0) || !isfinite(slope)) {       // fall back to projected steepest descent
        slope = 0.0;
        for (int k = lane; k < K; k += 32) {
          const double g = grad_s[k];
          const double v = (y_s[k] <= 0.0 && g >= 0.0) ? 0.0 : -g;
          d_s[k] = v;
          slope = fma(v, g, slope);
        }
        slope = warp_sum_f64(slope);
        if (lane == 0) si[5] = 1;
      } else if (lane == 0) {
        si[5] = 0;
      }
      __syncwarp();
      double tmax = CUDART_INF;
      int kbl = 0x7fffffff;
      for (int k = lane; k < K; k += 32) {
        const double v = d_s[k];
        if (v < 0.0) {
          const double tk = y_s[k] / (-v);
          if (tk < tmax) { tmax = tk; kbl = k; }
        }
      }
      const double tmin = warp_min_d(tmax);
      int cand_k = (tmax == tmin) ? kbl : 0x7fffffff;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) cand_k = min(cand_k, __shfl_xor_sync(0xffffffffu, cand_k, o));
      // Newton step (t = 1); steepest descent: one-dimensional Newton step t = -slope / (d^T H d)
      double t = 1.0;
      if (si[5]) {
        double dhd = 0.0;
        for (int a = lane; a < K; a += 32) {
          double row = 0.0;
          for (int b = 0; b < K; ++b) row = fma(h_sym(hred, nb, a, b), d_s[b], row);
          dhd = fma(d_s[a], row, dhd);
        }
        dhd = warp_sum_f64(dhd);
        t = (dhd > 0.0) ? -slope / dhd : ((tmin < CUDART_INF) ? tmin : 1.0);
      }
      const bool at_bound = t >= tmin;
      if (at_bound) t = tmin;
      for (int k = lane; k < K; k += 32) {
        double v = fmax(fma(t, d_s[k], y_s[k]), 0.0);
        if (at_bound && k == cand_k) v = 0.0;
        ytr_s[k] = v;
      }
      if (lane == 0) { sc[0] = t; sc[1] = slope; si[4] = (slope < 0.0) ? 0 : 1; }
    }
    wsync();
    PROF_MARK(4);
    if (si[4]) break;                                       // no descent direction left
    t_step = sc[0];
    slope0 = sc[1];
    have_dir = true;
    nbt = 0;
    pass(ytr_s);
    ++passes;
  }
  wsync();

  // ---- publish ----
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
        prof_s[7] += (unsigned long long)passes;
        PROF_MARK(10);
        for (int i = 0; i < kMasterProfSlots; ++i) p.prof[i] += prof_s[i];
      }
      DevState *st = p.st;
      st->K = K;
      st->m_iters = iters;
      st->m_passes = passes;
      st->m_hit_max = hit_max;
      st->n_hit_max += hit_max ? 1 : 0;
      st->m_restarts = 0;
      st->m_added = added;
      st->m_F = F;
      st->m_kkt = kkt;
      st->m_pg = pgmax;
      st->pg_iter_total += iters;
      st->pass_total += passes;
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

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
static size_t newton_fixed_smem(int32_t k_max, int32_t T, int32_t n_struct, int32_t n_red, int32_t lbuf_doubles) {
  return 128 + 128 + align_up((size_t)std::max(n_struct, 1) * sizeof(StructEntry), 128) + align_up((size_t)n_red * 8, 128) +
         align_up((size_t)lbuf_doubles * 8, 128) + (size_t)kNwtZThreads * 8 + 2 * align_up((size_t)(T + 4) * 8, 128) +
         align_up((size_t)(T + 8) * 2, 128);
}

NewtonLayout newton_layout(int32_t k_max, int32_t n_vox_pad, int32_t n_struct) {
  NewtonLayout L;
  L.nb_max = (k_max + 1 + 7) / 8;
  L.n_red = L.nb_max * (L.nb_max + 1) / 2 * 64 + 8;
  const int32_t lbuf = (k_max + 1) * (k_max + 2) / 2 + 8;
  // 227 KB opt-in maximum per CTA on sm_100; ~9 KB of static tables, 1 KB reserved by the system
  const size_t budget = (size_t)227 * 1024 - (size_t)10 * 1024;
  static const int32_t cand[] = {256, 192, 128, 96, 64, 32};
  for (int32_t T : cand) {
    const int32_t TP = T + 4;
    const int32_t stage = (int32_t)align_up((size_t)k_max * TP * 4, 128);
    const size_t fixed = newton_fixed_smem(k_max, T, n_struct, L.n_red, lbuf);
    if (fixed + (size_t)3 * stage > budget && T != 32) continue;
    int32_t stages = 2;
    while (stages < 6 && fixed + (size_t)(stages + 1) * stage <= budget) ++stages;
    L.T = T; L.TP = TP; L.stage_bytes = stage; L.n_stages = stages;
    L.smem = fixed + (size_t)stages * stage;
    break;
  }
  L.n_tiles = (n_vox_pad + L.T - 1) / L.T;
  L.tile_stride = (int64_t)k_max * L.TP;
  return L;
}

cudaError_t newton_configure(Ctx *c) {
  c->master_grid = std::min(c->n_sm, kMasterMaxGrid);
  const NewtonLayout &L = c->nwt;
  cudaError_t e = cudaFuncSetAttribute(k_master_newton, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);
  if (e != cudaSuccess) return e;
  int nbk = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nbk, k_master_newton, kMasterThreads, L.smem);
  if (e != cudaSuccess) return e;
  if (nbk < 1) return cudaErrorLaunchOutOfResources;
  return cudaSuccess;
}

cudaError_t launch_newton(Ctx *c, bool add_candidate) {
  const NewtonLayout &L = c->nwt;
  NewtonParams p{};
  p.A = c->d.A;
  p.n_vox_pad = c->n_vox_pad;
  p.T = L.T; p.TP = L.TP; p.tile_stride = L.tile_stride; p.n_tiles = L.n_tiles;
  p.n_stages = L.n_stages; p.stage_bytes = L.stage_bytes;
  p.n_red_cap = L.n_red;
  p.lbuf_doubles = (c->opt.k_max + 1) * (c->opt.k_max + 2) / 2 + 8;
  p.n_struct = std::max(c->n_struct, 1);
  p.sid = c->d.sid;
  p.vt = c->has_vt ? c->d.vt : nullptr;
  p.stab = c->d.stab;
  p.mz = c->d.mz;
  p.y = c->d.y;
  p.ll_part = c->d.ll_part;
  p.ll_result = c->d.ll_result;
  p.epoch = c->d.m_epoch;
  p.prof = (c->opt.reserved & 2) ? c->d.m_prof : nullptr;
  p.st = c->d.state;
  p.history = c->d.history;
  p.ap_beam = c->d.ap_beam;
  p.add_candidate = add_candidate ? 1 : 0;
  p.max_iter = c->opt.master_max_iter;
  p.k_max = c->opt.k_max;
  p.tol = c->opt.master_tol;
  void *args[] = {&p};
  return cudaLaunchCooperativeKernel((void *)k_master_newton, dim3(c->master_grid), dim3(kMasterThreads), args, L.smem,
                                     c->stream);
}

}  // namespace dao
