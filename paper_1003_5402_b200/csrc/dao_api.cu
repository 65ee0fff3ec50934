// dao_api.cu -- the extern "C" entry points of include/dao.h: argument marshalling, the
// column-generation driver (step 9) and the host<->device plumbing.
// Every arithmetic step runs in the kernels of dao_spmv.cu / dao_pricing.cu / dao_master.cu.
#include "dao_internal.cuh"

#include <math_constants.h>

#include <cstring>
#include <new>

using namespace dao;

static thread_local std::string g_last_error;

static dao_status fail(Ctx *c, dao_status st, const char *msg) {
  if (c) c->err = msg; else g_last_error = msg;
  return st;
}

#define API_CUDA(call)                                                                    \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                        \
      return DAO_E_CUDA;                                                                  \
    }                                                                                     \
  } while (0)

// ------------------------------------------------------------------------------------------
// small device helpers of the API layer (re-ordering between the caller's and the internal
// voxel order, pool upload)
// ------------------------------------------------------------------------------------------
namespace dao {

// tile_T > 0: `in` is in the tiled order of the Newton master (voxel i at slot i / n_tiles of tile i mod n_tiles)
template <typename T>
__global__ void k_to_user_order(int32_t n_vox_pad, const int32_t *__restrict__ perm, const T *__restrict__ in,
                                T *__restrict__ out, int32_t tile_T, int32_t n_tiles) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_vox_pad) return;
  const int32_t j = perm[i];
  if (j < 0) return;
  out[j] = tile_T > 0 ? in[(size_t)(i % n_tiles) * tile_T + (size_t)(i / n_tiles)] : in[i];
}

// 0/1 beamlet mask of pool aperture k (for dao_set_pool)
__global__ void k_pool_mask(int32_t k, int32_t n_bl, int32_t max_rows, const int32_t *__restrict__ bl_row,
                            const int32_t *__restrict__ row_beam, const int32_t *__restrict__ beam_row_ptr,
                            const int32_t *__restrict__ row_bl_ptr, const int32_t *__restrict__ ap_beam,
                            const int32_t *__restrict__ ap_left, const int32_t *__restrict__ ap_right,
                            float *__restrict__ xmask) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_bl) return;
  const int32_t r = bl_row[i], b = row_beam[r];
  float m = 0.f;
  if (b == ap_beam[k]) {
    const int32_t mm = r - beam_row_ptr[b], c = i - row_bl_ptr[r];
    m = (c >= ap_left[k * max_rows + mm] && c < ap_right[k * max_rows + mm]) ? 1.f : 0.f;
  }
  xmask[i] = m;
}

__global__ void k_set_pool_state(DevState *st, int32_t K) {
  st->K = K;
  st->cand_valid = 0;
  st->done = 0;
  // no master solve has been made for THIS pool: a duplicate candidate priced before one is reported as stalled,
  // never as a proof of optimality (reading S6 uses m_hit_max / m_kkt of the last solve)
  st->m_hit_max = 1;
  st->m_kkt = CUDART_INF;
}

static dao_status read_state(Ctx *c) {
  API_CUDA(cudaMemcpyAsync(c->h_state, c->d.state, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
  API_CUDA(cudaStreamSynchronize(c->stream));
  c->K = c->h_state->K;
  return DAO_OK;
}
// The same read-back in two halves: the copy is enqueued (and marked by an event) BEFORE further work goes into the
// stream, the host then waits for the event only -- the GPU keeps running what was enqueued behind the copy.
static dao_status enqueue_state_copy(Ctx *c) {
  API_CUDA(cudaMemcpyAsync(c->h_state, c->d.state, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
  API_CUDA(cudaEventRecord(c->ev_state, c->stream));
  return DAO_OK;
}
static dao_status wait_state_copy(Ctx *c) {
  API_CUDA(cudaEventSynchronize(c->ev_state));
  c->K = c->h_state->K;
  return DAO_OK;
}

// steps 1-3 at the current intensities
static dao_status enqueue_dose(Ctx *c) {
  API_CUDA(launch_intensity(c));
  API_CUDA(launch_spmv(c, kSpmvObjective, c->d.x, c->d.z));
  return DAO_OK;
}
// steps 4-6
static dao_status enqueue_pricing(Ctx *c) {
  API_CUDA(launch_spmv_t(c, c->d.g, c->d.w));
  API_CUDA(launch_pricing(c, c->d.w, c->d.row_bl_ptr, c->d.beam_row_ptr, c->n_rows, c->n_beams, c->d.left, c->d.right,
                          c->d.vstar, c->d.row_absmax, c->d.beam_price, c->d.beam_absmax, nullptr, true, c->max_row_len));
  return DAO_OK;
}
// step 7 (append + column) and step 8
static dao_status enqueue_column(Ctx *c) {
  API_CUDA(launch_append_candidate(c));
  API_CUDA(launch_spmv(c, kSpmvColumn, c->d.xmask, c->d.A));
  return DAO_OK;
}

}  // namespace dao

// ------------------------------------------------------------------------------------------
extern "C" {

void dao_default_options(dao_options *opt) {
  if (!opt) return;
  std::memset(opt, 0, sizeof(*opt));
  opt->k_max = 50;
  opt->master_max_iter = 2000;
  opt->master_tol = 1e-7;
  opt->price_tol = 1e-6;
  opt->master_method = 2;
  opt->master_ls_tol = 0.01;
  opt->sell_sigma = 0;
  opt->timers = 1;
  opt->mlc_mode = DAO_MLC_CONSECUTIVE;
}

dao_status dao_workspace_bytes(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                               dao_sizes *out) {
  dao_options o;
  if (opt) o = *opt; else dao_default_options(&o);
  return setup_sizes(D, mlc, s, &o, out, &g_last_error);
}

dao_status dao_create(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                      void *workspace, size_t workspace_bytes, void *scratch, size_t scratch_bytes,
                      void *cuda_stream, dao_ctx **out) {
  if (!out) return fail(nullptr, DAO_E_ARG, "null output pointer");
  *out = nullptr;
  Ctx *c = new (std::nothrow) Ctx();
  if (!c) return fail(nullptr, DAO_E_ALLOC, "out of host memory");
  if (opt) c->opt = *opt; else dao_default_options(&c->opt);
  c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  dao_status st = setup_build(c, D, mlc, s, workspace, workspace_bytes, scratch, scratch_bytes);
  if (st == DAO_OK) {
    cudaError_t e = cudaMallocHost(reinterpret_cast<void **>(&c->h_state), sizeof(DevState));
    for (int i = 0; i < 8 && e == cudaSuccess; ++i) e = cudaEventCreate(&c->ev[i]);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_state, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      c->err = std::string("host-side CUDA resources: ") + cudaGetErrorString(e);
      st = DAO_E_CUDA;
    } else {
      std::memset(c->h_state, 0, sizeof(DevState));
    }
  }
  if (st != DAO_OK) {
    g_last_error = c->err;
    if (c->h_state) cudaFreeHost(c->h_state);
    for (int i = 0; i < 8; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    if (c->ev_state) cudaEventDestroy(c->ev_state);
    delete c;
    return st;
  }
  *out = reinterpret_cast<dao_ctx *>(c);
  return DAO_OK;
}

dao_status dao_destroy(dao_ctx *ctx) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_OK;
  cudaStreamSynchronize(c->stream);
  if (c->h_state) cudaFreeHost(c->h_state);
  for (int i = 0; i < 8; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
  if (c->ev_state) cudaEventDestroy(c->ev_state);
  delete c;
  return DAO_OK;
}

const char *dao_last_error(const dao_ctx *ctx) {
  const Ctx *c = reinterpret_cast<const Ctx *>(ctx);
  return c ? c->err.c_str() : g_last_error.c_str();
}

dao_status dao_get_dims(const dao_ctx *ctx, dao_dims *out) {
  const Ctx *c = reinterpret_cast<const Ctx *>(ctx);
  if (!c || !out) return DAO_E_ARG;
  out->n_vox = c->n_vox; out->n_bl = c->n_bl; out->n_beams = c->n_beams; out->n_rows = c->n_rows;
  out->n_struct = c->n_struct; out->k_max = c->opt.k_max; out->nnz = c->nnz; out->sell_elems = c->sell_elems;
  out->sell_slice_rows = kSellC; out->sell_sigma = c->opt.sell_sigma; out->n_sm = c->n_sm; out->master_method = c->opt.master_method;
  return DAO_OK;
}

dao_status dao_reset(dao_ctx *ctx) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  API_CUDA(cudaMemsetAsync(c->d.state, 0, sizeof(DevState), c->stream));
  API_CUDA(cudaMemsetAsync(c->d.y, 0, DAO_MAX_APERTURES * sizeof(double), c->stream));
  API_CUDA(cudaMemsetAsync(c->d.x, 0, (size_t)c->n_bl * 4, c->stream));
  API_CUDA(cudaMemsetAsync(c->d.history, 0, (size_t)c->opt.k_max * sizeof(dao_iter_record), c->stream));
  API_CUDA(cudaStreamSynchronize(c->stream));
  c->K = 0;
  c->x_current = false;
  c->have_candidate = false;
  return DAO_OK;
}

dao_status dao_price(dao_ctx *ctx, dao_price_info *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  dao_status st = enqueue_dose(c);
  if (st == DAO_OK) st = enqueue_pricing(c);
  if (st == DAO_OK) st = read_state(c);
  if (st != DAO_OK) return st;
  const DevState &h = *c->h_state;
  c->have_candidate = h.cand_valid != 0;
  c->objective = h.F;
  if (out) {
    out->beam = h.cand_beam;
    out->converged = h.done == 1 ? 1 : 0;
    out->stalled = h.done == 2 ? 1 : 0;
    out->price = h.cand_price;
    out->objective = h.F;
    out->w_abs_max = h.w_abs_max;
    out->n_open_beamlets = h.cand_nopen;
    out->duplicate = h.cand_dup;
  }
  return DAO_OK;
}

static void fill_master_info(const Ctx *c, dao_master_info *out) {
  if (!out) return;
  const DevState &h = *c->h_state;
  out->n_apertures = h.K;
  out->n_pg_iter = h.m_iters;
  out->hit_max_iter = h.m_hit_max;
  out->n_restarts = h.m_restarts;
  out->objective = h.m_F;
  out->kkt_residual = h.m_kkt;
  out->pg_norm = h.m_pg;
  out->n_passes = h.m_passes;
  out->reserved = 0;
}

dao_status dao_solve_master(dao_ctx *ctx, dao_master_info *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  if (!c->have_candidate) return fail(c, DAO_E_STATE, "no pending candidate aperture (call dao_price first; pool full or already optimal)");
  dao_status st = enqueue_column(c);
  if (st != DAO_OK) return st;
  API_CUDA(launch_master(c, true));
  st = read_state(c);
  if (st != DAO_OK) return st;
  c->have_candidate = false;
  c->objective = c->h_state->m_F;
  fill_master_info(c, out);
  return DAO_OK;
}

dao_status dao_resolve_master(dao_ctx *ctx, dao_master_info *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  if (c->K <= 0) return fail(c, DAO_E_STATE, "empty aperture pool");
  API_CUDA(launch_master(c, false));
  dao_status st = read_state(c);
  if (st != DAO_OK) return st;
  c->objective = c->h_state->m_F;
  fill_master_info(c, out);
  return DAO_OK;
}

dao_status dao_run(dao_ctx *ctx, int32_t max_apertures, dao_run_info *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  if (max_apertures < 0 || max_apertures > c->opt.k_max) return fail(c, DAO_E_ARG, "max_apertures must be in [0, k_max]");
  dao_run_info info;
  std::memset(&info, 0, sizeof(info));
  const bool timers = c->opt.timers != 0;
  cudaEvent_t t0 = c->ev[7];
  // total time: ev[7] start, ev[6] of the last iteration / final evaluation as end
  API_CUDA(cudaEventRecord(t0, c->stream));
  dao_status st = read_state(c);
  if (st != DAO_OK) return st;
  const int64_t pg0 = c->h_state->pg_iter_total;
  const int32_t dup0 = c->h_state->n_duplicates;
  const int64_t pass0 = c->h_state->pass_total;
  const int32_t hit0 = c->h_state->n_hit_max;
  const int64_t launches0 = c->n_launches;
  double acc[6] = {0, 0, 0, 0, 0, 0};
  double pending[6] = {0, 0, 0, 0, 0, 0};   // times not yet written to a DAO_VEC_ITER_SECONDS row
  int n_resolve = 0;
  c->iter_seconds.clear();
  // Without timers the dose SpMV of the NEXT iteration (= the final dose evaluation when the loop ends) is enqueued
  // right behind the master, after the copy of the state block: the host reads the state while that SpMV runs, so
  // the GPU does not idle through the host round trip of the one synchronisation per iteration.
  bool dose_pending = false;
  while (c->K < max_apertures) {
    if (timers) API_CUDA(cudaEventRecord(c->ev[0], c->stream));
    if (!dose_pending) API_CUDA(launch_intensity(c));
    if (timers) API_CUDA(cudaEventRecord(c->ev[1], c->stream));
    if (!dose_pending) API_CUDA(launch_spmv(c, kSpmvObjective, c->d.x, c->d.z));
    dose_pending = false;
    if (timers) API_CUDA(cudaEventRecord(c->ev[2], c->stream));
    API_CUDA(launch_spmv_t(c, c->d.g, c->d.w));
    if (timers) API_CUDA(cudaEventRecord(c->ev[3], c->stream));
    API_CUDA(launch_pricing(c, c->d.w, c->d.row_bl_ptr, c->d.beam_row_ptr, c->n_rows, c->n_beams, c->d.left,
                            c->d.right, c->d.vstar, c->d.row_absmax, c->d.beam_price, c->d.beam_absmax, nullptr, true,
                            c->max_row_len));
    if (timers) API_CUDA(cudaEventRecord(c->ev[4], c->stream));
    st = enqueue_column(c);
    if (st != DAO_OK) return st;
    if (timers) API_CUDA(cudaEventRecord(c->ev[5], c->stream));
    API_CUDA(launch_master(c, true));
    if (timers) API_CUDA(cudaEventRecord(c->ev[6], c->stream));
    const int32_t k_before = c->K;
    if (timers) {
      st = read_state(c);               // the one host synchronisation of this iteration
    } else {
      st = enqueue_state_copy(c);
      if (st != DAO_OK) return st;
      st = enqueue_dose(c);             // x is the one the master just wrote (or left unchanged)
      if (st != DAO_OK) return st;
      dose_pending = true;
      st = wait_state_copy(c);          // the one host synchronisation of this iteration
    }
    if (st != DAO_OK) return st;
    ++info.n_iterations;
    if (timers) {
      for (int i = 0; i < 6; ++i) {
        float ms = 0.f;
        API_CUDA(cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        acc[i] += ms * 1e-3;
        pending[i] += ms * 1e-3;
      }
    }
    if (c->h_state->done == 2 && n_resolve < 2 && c->K > 0) {
      // stalled on a duplicate after an unconverged master (S6): solve the master further, then price again
      ++n_resolve;
      dose_pending = false;             // the re-solve changes x: the dose enqueued above is stale
      if (timers) API_CUDA(cudaEventRecord(c->ev[5], c->stream));
      API_CUDA(launch_master(c, false));
      if (timers) API_CUDA(cudaEventRecord(c->ev[6], c->stream));
      st = read_state(c);
      if (st != DAO_OK) return st;
      if (timers) {                     // the re-solve is master time of this call
        float ms = 0.f;
        API_CUDA(cudaEventElapsedTime(&ms, c->ev[5], c->ev[6]));
        acc[5] += ms * 1e-3;
        pending[5] += ms * 1e-3;
      }
      continue;
    }
    if (timers && c->K > k_before) {
      // one row per aperture ADDED, so that row i pairs with history record i of this call; an iteration that added
      // nothing (a stalled pricing and its re-solve) is charged to the next aperture's row
      for (int i = 0; i < 6; ++i) { c->iter_seconds.push_back(pending[i]); pending[i] = 0.0; }
    }
    if (c->h_state->done) { info.converged = c->h_state->done == 1 ? 1 : 0; info.stalled = c->h_state->done == 2 ? 1 : 0; break; }
    if (c->K == k_before) break;        // nothing was added (pool full)
  }
  // final dose evaluation of the returned plan (steps 1-3), unless it is already in the stream
  if (!dose_pending) {
    st = enqueue_dose(c);
    if (st != DAO_OK) return st;
  }
  API_CUDA(cudaEventRecord(c->ev[6], c->stream));
  st = read_state(c);
  if (st != DAO_OK) return st;
  float ms = 0.f;
  API_CUDA(cudaEventElapsedTime(&ms, t0, c->ev[6]));
  c->have_candidate = false;
  c->objective = c->h_state->F;
  info.n_apertures = c->K;
  info.n_duplicates = c->h_state->n_duplicates - dup0;
  info.n_pg_iter_total = c->h_state->pg_iter_total - pg0;
  info.n_passes_total = c->h_state->pass_total - pass0;
  info.n_hit_max_iter = c->h_state->n_hit_max - hit0;
  info.n_kernel_launches = (int32_t)(c->n_launches - launches0);
  info.objective = c->h_state->F;
  info.seconds_total = ms * 1e-3;
  info.seconds_intensity = acc[0]; info.seconds_spmv = acc[1]; info.seconds_spmv_t = acc[2];
  info.seconds_price = acc[3]; info.seconds_column = acc[4]; info.seconds_master = acc[5];
  if (out) *out = info;
  return DAO_OK;
}

dao_status dao_get_plan(dao_ctx *ctx, dao_plan *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !out) return DAO_E_ARG;
  dao_status st = read_state(c);
  if (st != DAO_OK) return st;
  const int32_t K = c->K, mr = c->max_rows_per_beam;
  std::vector<int32_t> beam((size_t)std::max(K, 1)), le((size_t)std::max(K, 1) * mr), ri((size_t)std::max(K, 1) * mr);
  std::vector<double> y((size_t)std::max(K, 1));
  if (K > 0) {
    API_CUDA(cudaMemcpyAsync(beam.data(), c->d.ap_beam, (size_t)K * 4, cudaMemcpyDeviceToHost, c->stream));
    API_CUDA(cudaMemcpyAsync(le.data(), c->d.ap_left, (size_t)K * mr * 4, cudaMemcpyDeviceToHost, c->stream));
    API_CUDA(cudaMemcpyAsync(ri.data(), c->d.ap_right, (size_t)K * mr * 4, cudaMemcpyDeviceToHost, c->stream));
    API_CUDA(cudaMemcpyAsync(y.data(), c->d.y, (size_t)K * 8, cudaMemcpyDeviceToHost, c->stream));
    API_CUDA(cudaStreamSynchronize(c->stream));
  }
  int32_t rows_used = 0;
  for (int32_t k = 0; k < K; ++k) rows_used += c->beam_row_ptr[beam[k] + 1] - c->beam_row_ptr[beam[k]];
  out->n_apertures = K;
  out->n_rows_used = rows_used;
  out->objective = c->objective;
  if (out->cap_apertures < K || out->cap_rows < rows_used) return fail(c, DAO_E_SHAPE, "dao_plan capacity too small");
  if (K > 0 && (!out->beam || !out->intensity || !out->ap_row_ptr || (rows_used > 0 && (!out->left || !out->right))))
    return fail(c, DAO_E_ARG, "null dao_plan array");
  int32_t pos = 0;
  if (out->ap_row_ptr) out->ap_row_ptr[0] = 0;
  for (int32_t k = 0; k < K; ++k) {
    const int32_t nr = c->beam_row_ptr[beam[k] + 1] - c->beam_row_ptr[beam[k]];
    out->beam[k] = beam[k];
    out->intensity[k] = (float)y[k];
    for (int32_t m = 0; m < nr; ++m) {
      out->left[pos + m] = le[(size_t)k * mr + m];
      out->right[pos + m] = ri[(size_t)k * mr + m];
    }
    pos += nr;
    out->ap_row_ptr[k + 1] = pos;
  }
  return DAO_OK;
}

dao_status dao_get_vector(dao_ctx *ctx, int32_t which, void *dst, dao_memspace mem) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !dst) return DAO_E_ARG;
  const void *src = nullptr;
  size_t bytes = 0;
  const int t = 256, gv = (c->n_vox_pad + t - 1) / t;
  switch (which) {
    case DAO_VEC_Z: src = c->d.z; bytes = (size_t)c->n_vox * 4; break;      // kept in the caller's order
    case DAO_VEC_G: src = c->d.g; bytes = (size_t)c->n_vox * 4; break;
    case DAO_VEC_MASTER_Z: {
      double *tmp = reinterpret_cast<double *>(c->d.io_scratch);
      k_to_user_order<double><<<gv, t, 0, c->stream>>>(c->n_vox_pad, c->d.perm, c->d.mz, tmp, c->nwt.T, c->nwt.n_tiles);
      API_CUDA(cudaGetLastError());
      src = tmp; bytes = (size_t)c->n_vox * 8;
      break;
    }
    case DAO_VEC_W: src = c->d.w; bytes = (size_t)c->n_bl * 4; break;
    case DAO_VEC_X: src = c->d.x; bytes = (size_t)c->n_bl * 4; break;
    case DAO_VEC_Y: src = c->d.y; bytes = (size_t)c->opt.k_max * 8; break;
    case DAO_VEC_VSTAR: src = c->d.vstar; bytes = (size_t)c->n_rows * 8; break;
    case DAO_VEC_LEFT: src = c->d.left; bytes = (size_t)c->n_rows * 4; break;
    case DAO_VEC_RIGHT: src = c->d.right; bytes = (size_t)c->n_rows * 4; break;
    case DAO_VEC_BEAM_PRICE: src = c->d.beam_price; bytes = (size_t)c->n_beams * 8; break;
    case DAO_VEC_MASTER_PHASES: src = c->d.m_prof; bytes = (size_t)kMasterProfSlots * 8; break;
    case DAO_VEC_HISTORY: src = c->d.history; bytes = (size_t)c->opt.k_max * sizeof(dao_iter_record); break;
    case DAO_VEC_ITER_SECONDS: {                          // host-resident: filled by dao_run from its CUDA events
      if (mem != DAO_MEM_HOST) return fail(c, DAO_E_ARG, "DAO_VEC_ITER_SECONDS is host data");
      double *out = reinterpret_cast<double *>(dst);
      const size_t n = (size_t)c->opt.k_max * 6;
      for (size_t i = 0; i < n; ++i) out[i] = i < c->iter_seconds.size() ? c->iter_seconds[i] : 0.0;
      return DAO_OK;
    }
    default: return fail(c, DAO_E_ARG, "unknown vector selector");
  }
  API_CUDA(cudaMemcpyAsync(dst, src, bytes, mem == DAO_MEM_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream));
  API_CUDA(cudaStreamSynchronize(c->stream));
  return DAO_OK;
}

dao_status dao_spmv(dao_ctx *ctx, const float *x_dev, float *z_dev) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !x_dev || !z_dev) return DAO_E_ARG;
  API_CUDA(launch_spmv(c, kSpmvPlainUserOrder, x_dev, z_dev));
  return DAO_OK;
}

dao_status dao_spmv_t(dao_ctx *ctx, const float *g_dev, float *w_dev) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !g_dev || !w_dev) return DAO_E_ARG;
  API_CUDA(launch_spmv_t(c, g_dev, w_dev));
  return DAO_OK;
}

dao_status dao_eval_x(dao_ctx *ctx, const float *x_dev, double *objective) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !x_dev) return DAO_E_ARG;
  API_CUDA(launch_spmv(c, kSpmvObjective, x_dev, c->d.z));
  dao_status st = read_state(c);
  if (st != DAO_OK) return st;
  if (objective) *objective = c->h_state->F;
  return DAO_OK;
}

dao_status dao_price_from_w(dao_ctx *ctx, const float *w_dev, const int32_t *row_bl_ptr_dev,
                            const int32_t *beam_row_ptr_dev, int32_t n_rows, int32_t n_beams, int32_t *left_dev,
                            int32_t *right_dev, double *vstar_dev, double *beam_price_dev, int32_t *best_dev) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c || !w_dev || !left_dev || !right_dev || !vstar_dev || !beam_price_dev || !best_dev) return DAO_E_ARG;
  const bool own = row_bl_ptr_dev == nullptr;
  if (!own && c->opt.mlc_mode != DAO_MLC_CONSECUTIVE)
    return fail(c, DAO_E_UNSUPPORTED, "caller-provided MLC tables are only supported with DAO_MLC_CONSECUTIVE");
  if (own) {
    if (beam_row_ptr_dev != nullptr) return fail(c, DAO_E_ARG, "pass both MLC tables or neither");
    row_bl_ptr_dev = c->d.row_bl_ptr; beam_row_ptr_dev = c->d.beam_row_ptr;
    n_rows = c->n_rows; n_beams = c->n_beams;
  } else if (!beam_row_ptr_dev || n_rows <= 0 || n_beams <= 0) {
    return fail(c, DAO_E_ARG, "bad MLC tables");
  }
  // row_absmax / beam_absmax scratch: the context's own arrays when they are large enough
  double *row_abs = c->d.row_absmax, *beam_abs = c->d.beam_absmax;
  if (!own && (n_rows > c->n_rows || n_beams > c->n_beams)) {
    // borrow the io scratch (>= 8 * (n_rows + n_beams) bytes required)
    const size_t cap = std::max<size_t>((size_t)c->n_vox_pad, (size_t)std::max(c->n_bl, c->n_rows)) + 64;
    if ((size_t)n_rows + (size_t)n_beams > cap) return fail(c, DAO_E_SHAPE, "MLC tables larger than the context's scratch");
    row_abs = reinterpret_cast<double *>(c->d.io_scratch);
    beam_abs = row_abs + n_rows;
  }
  API_CUDA(launch_pricing(c, w_dev, row_bl_ptr_dev, beam_row_ptr_dev, n_rows, n_beams, left_dev, right_dev, vstar_dev,
                          row_abs, beam_price_dev, beam_abs, best_dev, false, own ? c->max_row_len : -1));
  return DAO_OK;
}

dao_status dao_price_from_w_static(const float *w_dev, const int32_t *row_bl_ptr_dev, const int32_t *beam_row_ptr_dev,
                                   int32_t n_rows, int32_t n_beams, int32_t *left_dev, int32_t *right_dev,
                                   double *vstar_dev, double *beam_price_dev, int32_t *best_dev, void *cuda_stream) {
  // no context: failures are reported through dao_last_error(NULL) of the calling thread
  return price_from_w_static(w_dev, row_bl_ptr_dev, beam_row_ptr_dev, n_rows, n_beams, left_dev, right_dev, vstar_dev,
                             beam_price_dev, best_dev, static_cast<cudaStream_t>(cuda_stream), &g_last_error);
}

dao_status dao_set_pool(dao_ctx *ctx, int32_t n_apertures, const int32_t *beam, const int32_t *ap_row_ptr,
                        const int32_t *left, const int32_t *right, const double *y) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  const int32_t K = n_apertures, mr = c->max_rows_per_beam;
  if (K < 0 || K > c->opt.k_max) return fail(c, DAO_E_SHAPE, "n_apertures must be in [0, k_max]");
  if (K > 0 && (!beam || !ap_row_ptr || !left || !right)) return fail(c, DAO_E_ARG, "null pool array");
  std::vector<int32_t> le((size_t)std::max(K, 1) * mr, 0), ri((size_t)std::max(K, 1) * mr, 0);
  std::vector<double> yy(DAO_MAX_APERTURES, 0.0);
  std::vector<unsigned long long> hh((size_t)std::max(K, 1), 0ull);
  for (int32_t k = 0; k < K; ++k) {
    if (beam[k] < 0 || beam[k] >= c->n_beams) return fail(c, DAO_E_SHAPE, "aperture beam out of range");
    const int32_t r0 = c->beam_row_ptr[beam[k]], nr = c->beam_row_ptr[beam[k] + 1] - r0;
    if (ap_row_ptr[k + 1] - ap_row_ptr[k] != nr) return fail(c, DAO_E_SHAPE, "aperture row count does not match its beam");
    for (int32_t m = 0; m < nr; ++m) {
      const int32_t l = left[ap_row_ptr[k] + m], r = right[ap_row_ptr[k] + m];
      const int32_t n = c->row_bl_ptr[r0 + m + 1] - c->row_bl_ptr[r0 + m];
      if (l < 0 || r < l || r > n) return fail(c, DAO_E_SHAPE, "leaf positions out of range");
      le[(size_t)k * mr + m] = l; ri[(size_t)k * mr + m] = r;
      hh[k] += leaf_hash(m, l, r);
    }
    hh[k] += beam_hash(beam[k]);
    if (y) {
      if (!(y[k] >= 0.0)) return fail(c, DAO_E_ARG, "intensities must be >= 0");
      yy[k] = y[k];
    }
  }
  if (K > 0) {
    API_CUDA(cudaMemcpyAsync(c->d.ap_beam, beam, (size_t)K * 4, cudaMemcpyHostToDevice, c->stream));
    API_CUDA(cudaMemcpyAsync(c->d.ap_left, le.data(), (size_t)K * mr * 4, cudaMemcpyHostToDevice, c->stream));
    API_CUDA(cudaMemcpyAsync(c->d.ap_right, ri.data(), (size_t)K * mr * 4, cudaMemcpyHostToDevice, c->stream));
    API_CUDA(cudaMemcpyAsync(c->d.ap_hash, hh.data(), (size_t)K * 8, cudaMemcpyHostToDevice, c->stream));
  }
  API_CUDA(cudaMemcpyAsync(c->d.y, yy.data(), DAO_MAX_APERTURES * 8, cudaMemcpyHostToDevice, c->stream));
  k_set_pool_state<<<1, 1, 0, c->stream>>>(c->d.state, K);
  API_CUDA(cudaGetLastError());
  const int t = 128;
  for (int32_t k = 0; k < K; ++k) {
    k_pool_mask<<<(c->n_bl + t - 1) / t, t, 0, c->stream>>>(k, c->n_bl, mr, c->d.bl_row, c->d.row_beam, c->d.beam_row_ptr,
                                                            c->d.row_bl_ptr, c->d.ap_beam, c->d.ap_left, c->d.ap_right,
                                                            c->d.xmask);
    API_CUDA(cudaGetLastError());
    API_CUDA(launch_spmv(c, kSpmvColumn, c->d.xmask, c->d.A, nullptr, k));
  }
  API_CUDA(cudaStreamSynchronize(c->stream));   // le/ri/yy are stack-owned
  c->K = K;
  c->x_current = false;
  c->have_candidate = false;
  return DAO_OK;
}

dao_status dao_fmo_solve(dao_ctx *ctx, int32_t max_iter, double tol, int32_t warm_start, dao_fmo_info *out) {
  Ctx *c = reinterpret_cast<Ctx *>(ctx);
  if (!c) return DAO_E_ARG;
  if (max_iter < 0) return fail(c, DAO_E_ARG, "max_iter must be >= 0");
  c->x_current = false;               // x becomes the FMO variable
  c->have_candidate = false;          // the pending candidate was priced at a dose that is being overwritten
  return fmo_solve(c, max_iter, tol, warm_start != 0, out);
}

}  // extern "C"
