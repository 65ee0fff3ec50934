// dao_fmo.cu -- the FMO workload: min_{x >= 0} F(D x) over the beamlet intensities,
// "mathematically the same" model as DAO with single beamlets as columns, solved by "the same gradient
// projection method".  Per iteration, all on the device:
//   1  z = D x, F, pi = dF/dz     k_spmv_ring<objective>      (steps 2-3 of the hot path)
//   2  w = D^T pi                 k_spmvt + k_spmvt_finish    (step 4)
//   3  direction p: projected steepest descent -w on the free set {x_i > 0 or w_i < 0}, optionally
//      conjugated (Polak-Ribiere+), bent so that no bound cuts the ray before 2x the last step; slope phi'(0), t_max
//   4  dz = D p                   k_spmv_ring<plain>
//   5  step: root of phi'(t) = dz . pi(z + t dz) on [0, t_max] by safeguarded Newton on the
//      piecewise-linear phi' (passes over z, dz only, 2 x 4 V bytes, L2 resident)
//   6  x <- max(0, x + t p)
// No host round trip inside an iteration: every kernel reads its scalars from FmoState and returns at
// once when `done` is set; the host looks at the state every few iterations.  All sums are fp64 in a
// fixed order (block partials added in block order by the last block): bit-reproducible.
// The step rule is DESIGN.md reading S2 (the paper defers it to Men et al. 2009 / Bazaraa et al.).
#include "dao_internal.cuh"
#include "dao_ptx.cuh"

#include <math_constants.h>

#include <algorithm>

namespace dao {

constexpr int kFmoDirThreads = 1024;
constexpr int kFmoLsThreads = 256;
constexpr int kFmoRestartEvery = 200;   // steepest-descent restart of the conjugated direction

// block-wide reduction helpers for the single-CTA direction kernel (fixed order)
__device__ __forceinline__ double block_sum_d(double v, double *scratch) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = warp_sum_f64(v);
  __syncthreads();
  if (lane == 0) scratch[warp] = v;
  __syncthreads();
  double s = 0.0;
  for (int w = 0; w < nw; ++w) s += scratch[w];
  return s;
}
__device__ __forceinline__ double block_max_d(double v, double *scratch) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();
  if (lane == 0) scratch[warp] = v;
  __syncthreads();
  double s = scratch[0];
  for (int w = 1; w < nw; ++w) s = fmax(s, scratch[w]);
  return s;
}

// ---- step 3: search direction (one CTA; n_bl is at most a few 10^4) -------------------------------
__global__ void __launch_bounds__(kFmoDirThreads) k_fmo_direction(FmoState *__restrict__ fs, const DevState *__restrict__ st,
                                                                 int32_t n_bl, const float *__restrict__ x,
                                                                 const float *__restrict__ w, float *__restrict__ p,
                                                                 float *__restrict__ pgold, double tol, int32_t max_iter,
                                                                 int32_t method) {
  __shared__ double scratch[kFmoDirThreads / 32];
  if (fs->done) return;
  const int tid = threadIdx.x;
  const double F = st->F;
  // pass 1: projected steepest descent pg, its norms, the Polak-Ribiere sums, free-set change
  double pg_max = 0.0, x_max = 1.0, kkt = 0.0, num = 0.0, den = 0.0;
  const double t_ref = 0.5 * fs->t_est;
  for (int i = tid; i < n_bl; i += kFmoDirThreads) {
    const double xi = (double)x[i], wi = (double)w[i], po = (double)pgold[i];
    const bool fr = (xi > 0.0) || (wi < 0.0);
    const double pg = fr ? -wi : 0.0;
    // stationarity measure |x - P(x - t_ref w)| / t_ref (t_ref = last accepted step): a positive variable
    // with w_i > 0 that sits closer to its bound than one step counts with x_i / t_ref, not with w_i
    double m = fabs(pg);
    if (wi > 0.0 && t_ref > 0.0) m = fmin(m, xi / t_ref);
    pg_max = fmax(pg_max, m);
    x_max = fmax(x_max, xi);
    kkt = fmax(kkt, (xi > 0.0) ? m : fmax(-wi, 0.0));
    num = fma(pg, pg - po, num);
    den = fma(po, po, den);
  }
  pg_max = block_max_d(pg_max, scratch);
  x_max = block_max_d(x_max, scratch);
  kkt = block_max_d(kkt, scratch);
  num = block_sum_d(num, scratch);
  den = block_sum_d(den, scratch);
  const int iters = fs->iters;
  // w is an fp32 vector: once F stops decreasing beyond fp64 rounding for 4 iterations in a row the
  // iterate sits at the resolution of the arithmetic and counts as converged (converged = 2)
  // (a step that was cut at a bound does not count: it can be arbitrarily short)
  const bool flat = iters > 0 && !fs->force_restart && fabs(fs->F_prev - F) <= 1e-13 * fabs(F);
  const int stall = flat ? fs->stall + 1 : 0;
  const bool conv = pg_max * x_max <= tol * fmax(F, 1e-300) || stall >= 4;
  const bool stop = conv || iters >= max_iter;
  if (stop) {
    __syncthreads();
    if (tid == 0) {
      fs->F = F; fs->pg_max = pg_max; fs->kkt = kkt; fs->x_max = x_max;
      fs->converged = conv ? (stall >= 4 ? 2 : 1) : 0; fs->hit_max = conv ? 0 : 1;
      __threadfence();
      fs->done = 1;
    }
    return;
  }
  bool restart = fs->force_restart || method == 0 || fs->since_restart >= kFmoRestartEvery || !(den > 0.0);
  double beta = 0.0;
  if (!restart) beta = fmax(num / den, 0.0);
  if (beta == 0.0) restart = true;
  // Bending (projection-arc idea, Bertsekas): a component that would cross its bound before t_est
  // is slowed down so that it reaches 0 exactly at t_est.  The first bound on the ray is then never
  // closer than t_est, and many variables can land on their bounds in one step, instead of the
  // ray being cut at the first of thousands of bounds.  The bent direction is still a descent
  // direction (checked), so the method stays a feasible descent method with an exact line search.
  const double t_est = fs->t_est;
  // pass 2: conjugated direction (fp32-representable), its slope and feasibility
  double slope = 0.0;
  for (int i = tid; i < n_bl; i += kFmoDirThreads) {
    const double xi = (double)x[i], wi = (double)w[i];
    const bool fr = (xi > 0.0) || (wi < 0.0);
    double v = fr ? -wi : 0.0;
    if (!restart && v != 0.0) v = fma(beta, (double)p[i], v);
    if (v < 0.0 && !(xi > 0.0)) v = fr ? -wi : 0.0;          // a variable at its bound may only move inwards
    if (v < 0.0 && t_est > 0.0 && fma(t_est, v, xi) < 0.0) v = -xi / t_est;
    v = (double)(float)v;
    slope = fma(v, wi, slope);
  }
  slope = block_sum_d(slope, scratch);
  if (!restart && !(slope < 0.0)) restart = true, beta = 0.0;
  // pass 3: write p, pgold; slope, t_max and the blocking variable
  slope = 0.0;
  double tmax = CUDART_INF;
  for (int i = tid; i < n_bl; i += kFmoDirThreads) {
    const double xi = (double)x[i], wi = (double)w[i];
    const bool fr = (xi > 0.0) || (wi < 0.0);
    const double pg = fr ? -wi : 0.0;
    double v = pg;
    if (!restart && v != 0.0) v = fma(beta, (double)p[i], v);
    if (v < 0.0 && !(xi > 0.0)) v = pg;
    if (v < 0.0 && t_est > 0.0 && fma(t_est, v, xi) < 0.0) v = -xi / t_est;
    const float vf = (float)v;
    p[i] = vf;
    pgold[i] = (float)pg;
    slope = fma((double)vf, wi, slope);
    if (vf < 0.f) tmax = fmin(tmax, xi / (-(double)vf));
  }
  slope = block_sum_d(slope, scratch);
  const double tmin = -block_max_d(-tmax, scratch);
  // smallest index attaining t_max
  int ib = 0x7fffffff;
  for (int i = tid; i < n_bl; i += kFmoDirThreads) {
    const float vf = p[i];
    if (vf < 0.f && (double)x[i] / (-(double)vf) == tmin) { ib = i; break; }
  }
  const double ibm = -block_max_d(-(double)ib, scratch);
  if (tid == 0) {
    fs->F = F; fs->pg_max = pg_max; fs->kkt = kkt; fs->x_max = x_max;
    fs->F_prev = F; fs->stall = stall;
    fs->slope0 = slope; fs->tmax = tmin; fs->ib = (int)ibm;
    fs->lo = 0.0; fs->slo = slope; fs->hi = CUDART_INF; fs->shi = 0.0;
    fs->t = 0.0; fs->ls_done = (slope < 0.0) ? 0 : 1;        // no descent left: zero step
    fs->at_bound = 0;
    if (restart) { fs->restarts += 1; fs->since_restart = 0; } else { fs->since_restart += 1; }
    fs->force_restart = 0;
  }
}

// ---- step 5: line search on (z, dz) --------------------------------------------------------------
// One pass: s1 = phi'(t) = sum dz_j pi_j(z_j + t dz_j), s2 = phi''(t) = sum 2 c_j dz_j^2 with c_j the
// weight of the active penalty branch.  INIT evaluates at t = 0 and proposes the Newton step
// -phi'(0) / phi''(0) (exact while no voxel changes branch), clipped to t_max; EVAL evaluates at the
// trial step and either accepts it (|phi'(t)| <= ls_tol |phi'(0)|, or still descending at the bound) or
// refines the bracket (Newton from the current point, regula falsi / bisection as safeguards).
struct FmoLsParams {
  FmoState *fs;
  int32_t n_vox_pad;
  const int32_t *perm;       // internal -> caller voxel (z is kept in the caller's order)
  const uint8_t *sid;
  const StructEntry *stab;
  const float *vt;
  const float *z;
  const float *dz;           // internal order
  double *part;              // [2 * grid]
  double ls_tol;
  int32_t last;              // 1: the last evaluation of this iteration -- settle on a safe step
};

template <bool INIT>
__global__ void __launch_bounds__(kFmoLsThreads) k_fmo_ls(FmoLsParams q) {
  __shared__ double red[2][kFmoLsThreads / 32];
  __shared__ bool is_last;
  FmoState *fs = q.fs;
  if (fs->done || fs->ls_done) return;
  const double t = INIT ? 0.0 : fs->t;
  double s1 = 0.0, s2 = 0.0;
  for (int i = blockIdx.x * kFmoLsThreads + threadIdx.x; i < q.n_vox_pad; i += gridDim.x * kFmoLsThreads) {
    const int s = q.sid[i];
    if (s == kNoStruct) continue;
    const int32_t j = q.perm[i];
    if (j < 0) continue;
    StructEntry e = q.stab[s];
    if (q.vt) e.tm = e.tp = (double)q.vt[i];
    const double dz = (double)q.dz[i];
    const double zz = fma(t, dz, (double)q.z[j]);
    const double u = fmax(e.tm - zz, 0.0), o = fmax(zz - e.tp, 0.0);
    const double gv = -2.0 * e.a * u + 2.0 * e.b * o;
    const double c = (u > 0.0 ? e.a : 0.0) + (o > 0.0 ? e.b : 0.0);
    s1 = fma(dz, gv, s1);
    s2 = fma(2.0 * c * dz, dz, s2);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  s1 = warp_sum_f64(s1);
  s2 = warp_sum_f64(s2);
  if (lane == 0) { red[0][warp] = s1; red[1][warp] = s2; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < kFmoLsThreads / 32; ++w) { a += red[0][w]; b += red[1][w]; }
    q.part[2 * blockIdx.x] = a;
    q.part[2 * blockIdx.x + 1] = b;
    __threadfence();
    is_last = atomicAdd(&fs->ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last || warp != 0) return;
  __threadfence();
  double c1 = 0.0, c2 = 0.0;
  for (int b = lane; b < (int)gridDim.x; b += 32) { c1 += __ldcg(q.part + 2 * b); c2 += __ldcg(q.part + 2 * b + 1); }
  c1 = warp_sum_f64(c1);
  c2 = warp_sum_f64(c2);
  if (lane != 0) return;
  fs->ticket = 0u;
  fs->ls_evals += 1;
  const double slope0 = fs->slope0, tmax = fs->tmax;
  if (INIT) {
    double tn = (c2 > 0.0) ? (-slope0 / c2) : ((tmax < CUDART_INF) ? tmax : 1.0);
    if (tn > tmax) tn = tmax;
    fs->t = tn; fs->c1 = slope0; fs->c2 = c2;
    return;
  }
  fs->c1 = c1; fs->c2 = c2;
  double lo = fs->lo, slo = fs->slo, hi = fs->hi, shi = fs->shi;
  if (fabs(c1) <= q.ls_tol * fabs(slope0)) { fs->ls_done = 1; return; }
  if (c1 < 0.0 && t >= tmax) { fs->ls_done = 1; fs->at_bound = 1; return; }
  double tn;
  if (c1 < 0.0) {
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
  if (q.last) {
    // out of evaluations: a point with phi' < 0 is a guaranteed decrease (phi convex); without one,
    // the secant root of the bracket
    if (hi < CUDART_INF) tn = (lo > 0.0) ? lo : lo + (hi - lo) * (-slo) / (shi - slo);
    else tn = t;
    fs->ls_done = 1;
    fs->at_bound = (tn >= tmax && c1 < 0.0) ? 1 : 0;
  }
  fs->lo = lo; fs->slo = slo; fs->hi = hi; fs->shi = shi;
  fs->t = tn;
}

// ---- step 6: x <- max(0, x + t p) ----------------------------------------------------------------
__global__ void k_fmo_update(FmoState *__restrict__ fs, int32_t n_bl, float *__restrict__ x, const float *__restrict__ p) {
  if (fs->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const double t = fs->t;
  const int at_bound = fs->at_bound, ib = fs->ib;
  if (i < n_bl) {
    double v = fma(t, (double)p[i], (double)x[i]);
    if (v < 0.0 || (at_bound && i == ib)) v = 0.0;
    x[i] = (float)v;
  }
}
__global__ void k_fmo_reset(FmoState *fs, int keep_horizon) {
  const double te = keep_horizon ? fs->t_est : 0.0;      // a warm start keeps the step scale of the last solve
  *fs = FmoState{};
  fs->t_est = te;
}
__global__ void k_fmo_advance(FmoState *fs) {
  if (fs->done) return;
  fs->iters += 1;
  fs->force_restart = fs->at_bound;
  if (fs->t > 0.0) fs->t_est = 2.0 * fs->t;
}

// ---- host driver ----------------------------------------------------------------------------------
#define FMO_CUDA(call)                                                                    \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                        \
      return DAO_E_CUDA;                                                                  \
    }                                                                                     \
  } while (0)

constexpr int kFmoLsEvals = 5;        // evaluations of phi'(t) per iteration after the Newton proposal
constexpr int kFmoCheckEvery = 8;     // iterations between two host looks at the state

dao_status fmo_solve(Ctx *c, int32_t max_iter, double tol, bool warm_start, dao_fmo_info *out) {
  FmoState *fs = c->d.fmo_state;
  const int32_t *skip = &fs->done;
  k_fmo_reset<<<1, 1, 0, c->stream>>>(fs, warm_start ? 1 : 0);
  FMO_CUDA(cudaGetLastError());
  FMO_CUDA(cudaMemsetAsync(c->d.fmo_p, 0, (size_t)c->n_bl * 4, c->stream));
  FMO_CUDA(cudaMemsetAsync(c->d.fmo_pgold, 0, (size_t)c->n_bl * 4, c->stream));
  if (!warm_start) FMO_CUDA(cudaMemsetAsync(c->d.x, 0, (size_t)c->n_bl * 4, c->stream));
  if (!(tol > 0.0)) tol = c->opt.master_tol;
  FmoLsParams q{};
  q.fs = fs; q.n_vox_pad = c->n_vox_pad; q.perm = c->d.perm; q.sid = c->d.sid; q.stab = c->d.stab;
  q.vt = c->has_vt ? c->d.vt : nullptr; q.z = c->d.z; q.dz = c->d.fmo_dz; q.part = c->d.fmo_part;
  q.ls_tol = c->opt.master_ls_tol;
  int ls_grid = std::min(kFmoLsGridMax, std::max(1, std::min(c->n_sm * 4, (c->n_vox_pad + kFmoLsThreads - 1) / kFmoLsThreads)));
  const int ug = (c->n_bl + 255) / 256;
  cudaEvent_t e0 = c->ev[0], e1 = c->ev[1];
  FMO_CUDA(cudaEventRecord(e0, c->stream));
  FmoState h{};
  // The loop bound covers the iteration that detects the cap / convergence (it does no update).
  for (int32_t it = 0; it <= max_iter; ++it) {
    FMO_CUDA(launch_spmv(c, kSpmvObjective, c->d.x, c->d.z, skip));
    FMO_CUDA(launch_spmv_t(c, c->d.g, c->d.w, skip));
    k_fmo_direction<<<1, kFmoDirThreads, 0, c->stream>>>(fs, c->d.state, c->n_bl, c->d.x, c->d.w, c->d.fmo_p,
                                                         c->d.fmo_pgold, tol, max_iter, c->opt.master_method);
    FMO_CUDA(cudaGetLastError());
    FMO_CUDA(launch_spmv(c, kSpmvPlain, c->d.fmo_p, c->d.fmo_dz, skip));
    q.last = 0;
    k_fmo_ls<true><<<ls_grid, kFmoLsThreads, 0, c->stream>>>(q);
    for (int e = 0; e < kFmoLsEvals; ++e) {
      q.last = (e == kFmoLsEvals - 1) ? 1 : 0;
      k_fmo_ls<false><<<ls_grid, kFmoLsThreads, 0, c->stream>>>(q);
    }
    k_fmo_update<<<ug, 256, 0, c->stream>>>(fs, c->n_bl, c->d.x, c->d.fmo_p);
    k_fmo_advance<<<1, 1, 0, c->stream>>>(fs);
    FMO_CUDA(cudaGetLastError());
    if ((it + 1) % kFmoCheckEvery == 0 || it == max_iter) {
      FMO_CUDA(cudaMemcpyAsync(&h, fs, sizeof(FmoState), cudaMemcpyDeviceToHost, c->stream));
      FMO_CUDA(cudaStreamSynchronize(c->stream));
      if (h.done) break;
    }
  }
  FMO_CUDA(cudaEventRecord(e1, c->stream));
  FMO_CUDA(cudaMemcpyAsync(&h, fs, sizeof(FmoState), cudaMemcpyDeviceToHost, c->stream));
  FMO_CUDA(cudaStreamSynchronize(c->stream));
  float ms = 0.f;
  FMO_CUDA(cudaEventElapsedTime(&ms, e0, e1));
  c->objective = h.F;
  if (out) {
    out->n_iter = h.iters; out->converged = h.converged; out->hit_max_iter = h.hit_max;
    out->n_restarts = h.restarts; out->n_ls_evals = h.ls_evals; out->reserved = 0;
    out->objective = h.F; out->kkt_residual = h.kkt; out->pg_norm = h.pg_max; out->seconds = ms * 1e-3;
  }
  return DAO_OK;
}

}  // namespace dao
