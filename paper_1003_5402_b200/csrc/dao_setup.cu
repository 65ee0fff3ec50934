// dao_setup.cu -- dao_workspace_bytes / dao_create: validation, upload, and the one-time
// construction of the device layouts:
//   * sliced-ELL copy of D in an internal voxel order (rows sorted by length, by default over
//     the whole matrix, so that the 32-row slices carry ~0 % padding),
//   * explicit CSR of D^T (PAPER.md:171 rebuilds the transpose every iteration with Thrust; D is
//     fixed here, so it is built once) by a stable LSD radix sort on the column index,
//   * chunk tables of the transposed SpMV, MLC lookup tables, the per-structure penalty table
//     alpha_s/|v_s|, beta_s/|v_s|, T_s^-, T_s^+ of eq. (9)-(10).
#include "dao_internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

namespace dao {

// ------------------------------------------------------------------------------------------
// host-side layout decisions
// ------------------------------------------------------------------------------------------
struct HostLayout {
  int32_t n_vox_pad = 0, n_slices = 0;
  int64_t sell_elems = 0;
  std::vector<int32_t> perm;          // [n_vox_pad] internal -> caller (-1 padding)
  std::vector<int32_t> inv_perm;      // [n_vox]
  std::vector<uint32_t> slice_off;    // [n_slices+1]
};

// 0 = library default = one window over all rows (global sort by length: no padding beyond the
// 32-row slice granularity; z and g are scattered to the caller's order, so nothing else depends on it)
static int effective_sigma(const dao_options *opt, int32_t n_vox) {
  return opt->sell_sigma > 0 ? opt->sell_sigma : std::max(n_vox, 1);
}

static dao_status make_layout(const int32_t *row_ptr, int32_t n_vox, int sigma, HostLayout *L, std::string *err) {
  L->n_vox_pad = (int32_t)align_up((size_t)std::max(n_vox, 1), 128);
  L->n_slices = L->n_vox_pad / kSellC;
  L->perm.assign(L->n_vox_pad, -1);
  L->inv_perm.assign(n_vox, 0);
  std::iota(L->perm.begin(), L->perm.begin() + n_vox, 0);
  if (sigma >= n_vox && n_vox > 1) {
    // one window: stable counting sort by descending row length
    int32_t max_len = 0;
    for (int32_t j = 0; j < n_vox; ++j) max_len = std::max(max_len, row_ptr[j + 1] - row_ptr[j]);
    std::vector<int32_t> start((size_t)max_len + 2, 0);
    for (int32_t j = 0; j < n_vox; ++j) ++start[(size_t)(max_len - (row_ptr[j + 1] - row_ptr[j])) + 1];
    for (size_t b = 1; b < start.size(); ++b) start[b] += start[b - 1];
    for (int32_t j = 0; j < n_vox; ++j) L->perm[start[(size_t)(max_len - (row_ptr[j + 1] - row_ptr[j]))]++] = j;
  } else if (sigma > 1) {
    for (int32_t s = 0; s < n_vox; s += sigma) {
      const int32_t e = std::min(n_vox, s + sigma);
      std::stable_sort(L->perm.begin() + s, L->perm.begin() + e, [&](int32_t a, int32_t b) {
        return (row_ptr[a + 1] - row_ptr[a]) > (row_ptr[b + 1] - row_ptr[b]);
      });
    }
  }
  for (int32_t i = 0; i < n_vox; ++i) L->inv_perm[L->perm[i]] = i;
  L->slice_off.assign(L->n_slices + 1, 0);
  int64_t total = 0;
  for (int32_t s = 0; s < L->n_slices; ++s) {
    int32_t mx = 0;
    for (int r = 0; r < kSellC; ++r) {
      const int32_t j = L->perm[s * kSellC + r];
      if (j >= 0) mx = std::max(mx, row_ptr[j + 1] - row_ptr[j]);
    }
    L->slice_off[s] = (uint32_t)total;
    total += (int64_t)mx * kSellC;
    if (total >= ((int64_t)1 << 32) - 64) {
      *err = "sliced-ELL copy of D would exceed 2^32 elements";
      return DAO_E_UNSUPPORTED;
    }
  }
  L->slice_off[L->n_slices] = (uint32_t)total;
  L->sell_elems = total;
  return DAO_OK;
}

// ------------------------------------------------------------------------------------------
// workspace carving (one function decides every offset; called with base = nullptr for sizing)
// ------------------------------------------------------------------------------------------
struct Carver {
  unsigned char *base;
  size_t off = 0;
  template <typename T>
  T *take(size_t n) {
    off = align_up(off, 256);
    T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

struct Dims {
  int32_t n_vox, n_bl, n_beams, n_rows, k_max, max_rows;
  int32_t chain_states;        // (W+1)^2 leaf states per row of the chain pricing modes, 0 otherwise
  int64_t nnz;
  int32_t master_method;
  int32_t n_struct;
};

// layout of the dose block and of the grid-reduction slots, decided by the master method alone
static NewtonLayout layout_of_master(const Dims &dm, int32_t n_vox_pad) {
  if (dm.master_method >= 2) return newton_layout(dm.k_max, n_vox_pad, dm.n_struct, dm.master_method == 3);
  return NewtonLayout{};
}

static int64_t tchunks_of(int64_t nnz) { return (nnz + kTChunk - 1) / kTChunk; }

static void carve_workspace(Carver &cv, const Dims &dm, const HostLayout &L, DevPtrs *d, int n_sm) {
  const size_t vp = (size_t)L.n_vox_pad;
  const int64_t ntc = tchunks_of(dm.nnz);
  d->sell_col = cv.take<int32_t>((size_t)L.sell_elems + 64);
  d->sell_val = cv.take<float>((size_t)L.sell_elems + 64);
  d->slice_off = cv.take<uint32_t>((size_t)L.n_slices + 1);
  d->perm = cv.take<int32_t>(vp);
  d->inv_perm = cv.take<int32_t>((size_t)dm.n_vox);
  d->sid = cv.take<uint8_t>(vp);
  d->stab = cv.take<StructEntry>(256);
  d->vt = cv.take<float>(vp);
  d->t_ptr = cv.take<int32_t>((size_t)dm.n_bl + 2);
  d->t_row = cv.take<int32_t>((size_t)ntc * kTChunk + 64);
  d->t_val = cv.take<float>((size_t)ntc * kTChunk + 64);
  d->t_first_row = cv.take<int32_t>((size_t)ntc + 1);
  d->t_seg_base = cv.take<int32_t>((size_t)ntc + 2);
  d->t_segsum = cv.take<double>((size_t)ntc + (size_t)dm.n_bl + 2);
  d->beam_row_ptr = cv.take<int32_t>((size_t)dm.n_beams + 1);
  d->row_bl_ptr = cv.take<int32_t>((size_t)dm.n_rows + 1);
  d->bl_row = cv.take<int32_t>((size_t)dm.n_bl);
  d->row_beam = cv.take<int32_t>((size_t)dm.n_rows);
  d->row_col0 = cv.take<int32_t>((size_t)dm.n_rows);
  d->chain_from = cv.take<int32_t>((size_t)dm.n_rows * (size_t)dm.chain_states + 4);
  d->x = cv.take<float>((size_t)dm.n_bl);
  d->xmask = cv.take<float>((size_t)dm.n_bl);
  d->z = cv.take<float>(vp);
  d->g = cv.take<float>(vp);
  d->w = cv.take<float>((size_t)dm.n_bl);
  d->f_part = cv.take<double>((size_t)n_sm * 8 + 64);
  d->vstar = cv.take<double>((size_t)dm.n_rows);
  d->left = cv.take<int32_t>((size_t)dm.n_rows);
  d->right = cv.take<int32_t>((size_t)dm.n_rows);
  d->row_absmax = cv.take<double>((size_t)dm.n_rows);
  d->beam_price = cv.take<double>((size_t)dm.n_beams);
  d->beam_absmax = cv.take<double>((size_t)dm.n_beams);
  d->ap_beam = cv.take<int32_t>((size_t)dm.k_max);
  d->ap_hash = cv.take<unsigned long long>((size_t)dm.k_max);
  d->ap_left = cv.take<int32_t>((size_t)dm.k_max * dm.max_rows);
  d->ap_right = cv.take<int32_t>((size_t)dm.k_max * dm.max_rows);
  const NewtonLayout nl = layout_of_master(dm, L.n_vox_pad);
  d->A = cv.take<float>(nl.T ? (size_t)nl.n_tiles * (size_t)nl.tile_stride : (size_t)dm.k_max * vp);
  d->y = cv.take<double>((size_t)DAO_MAX_APERTURES);
  d->mz = cv.take<double>(nl.T ? (size_t)nl.n_tiles * (size_t)nl.T : vp);   // the Newton master keeps it in the tiled order
  d->mdz = cv.take<double>(vp);
  {
    const size_t g = (size_t)std::min(n_sm * kMasterCtasPerSm, kMasterMaxGrid);
    const size_t stride = nl.T ? (size_t)nl.n_red : (size_t)kMaxRedux;
    d->ll_part = cv.take<uint4>(2 * g * stride);
    d->ll_result = cv.take<uint4>(2 * stride);
  }
  d->m_epoch = cv.take<uint32_t>(64);
  d->m_prof = cv.take<unsigned long long>(kMasterProfSlots);
  d->fmo_p = cv.take<float>((size_t)dm.n_bl);
  d->fmo_pgold = cv.take<float>((size_t)dm.n_bl);
  d->fmo_dz = cv.take<float>(vp);
  d->fmo_part = cv.take<double>(2 * (size_t)kFmoLsGridMax);
  d->fmo_state = cv.take<FmoState>(1);
  d->history = cv.take<dao_iter_record>((size_t)dm.k_max);
  d->state = cv.take<DevState>(1);
  d->io_scratch = cv.take<double>(std::max<size_t>(vp, (size_t)std::max(dm.n_bl, dm.n_rows)) + 64);
}

// create-time scratch
struct ScratchPtrs {
  int32_t *row_ptr, *col, *vs;
  float *val, *vt;
  int32_t *keyA, *rowA, *keyB, *rowB;
  float *valA, *valB;
  int32_t *tile_hist;
  int32_t *scan_sums;      // block totals of the multi-CTA scan
  int32_t *flags;
};
constexpr int kRadixThreads = 256, kRadixItems = 16, kRadixTile = kRadixThreads * kRadixItems;
constexpr int kScanChunk = 16384;    // elements per CTA of the multi-CTA scan

static void carve_scratch(Carver &cv, const Dims &dm, bool host_inputs, ScratchPtrs *s) {
  const size_t nz = (size_t)dm.nnz + 64;
  if (host_inputs) {
    s->row_ptr = cv.take<int32_t>((size_t)dm.n_vox + 1);
    s->col = cv.take<int32_t>(nz);
    s->val = cv.take<float>(nz);
    s->vs = cv.take<int32_t>((size_t)dm.n_vox);
    s->vt = cv.take<float>((size_t)dm.n_vox);
  } else {
    s->row_ptr = s->col = s->vs = nullptr;
    s->val = s->vt = nullptr;
  }
  s->keyA = cv.take<int32_t>(nz);
  s->rowA = cv.take<int32_t>(nz);
  s->valA = cv.take<float>(nz);
  s->keyB = cv.take<int32_t>(nz);
  s->rowB = cv.take<int32_t>(nz);
  s->valB = cv.take<float>(nz);
  const size_t n_tiles = ((size_t)dm.nnz + kRadixTile - 1) / kRadixTile;
  s->tile_hist = cv.take<int32_t>(256 * n_tiles + 1024);
  s->scan_sums = cv.take<int32_t>((256 * n_tiles) / kScanChunk + 1024);
  s->flags = cv.take<int32_t>(260);
}

// ------------------------------------------------------------------------------------------
// argument checks shared by sizes / create (host only)
// ------------------------------------------------------------------------------------------
static dao_status check_args(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                             Dims *dm, std::string *err) {
  if (!D || !mlc || !s || !opt) { *err = "null argument"; return DAO_E_ARG; }
  if (D->n_vox <= 0 || D->n_bl <= 0 || D->nnz < 0) { *err = "n_vox, n_bl must be positive and nnz >= 0"; return DAO_E_ARG; }
  if (D->nnz >= ((int64_t)1 << 31) - 2 * kTChunk) { *err = "nnz >= 2^31"; return DAO_E_UNSUPPORTED; }
  if (!D->row_ptr || (D->nnz > 0 && (!D->col_idx || !D->val))) { *err = "null CSR array"; return DAO_E_ARG; }
  if (D->mem != DAO_MEM_HOST && D->mem != DAO_MEM_DEVICE) { *err = "bad dao_csr.mem"; return DAO_E_ARG; }
  if (mlc->n_beams <= 0 || mlc->n_rows <= 0 || !mlc->beam_row_ptr || !mlc->row_bl_ptr) {
    *err = "bad MLC description"; return DAO_E_ARG;
  }
  if (s->n_struct < 0 || !s->vox_struct) { *err = "bad structure description"; return DAO_E_ARG; }
  if (s->n_struct > kMaxStruct) { *err = "more than 255 structures"; return DAO_E_UNSUPPORTED; }
  if (s->n_struct > 0 && (!s->t_under || !s->w_under || !s->t_over || !s->w_over)) {
    *err = "null structure table"; return DAO_E_ARG;
  }
  for (int i = 0; i < s->n_struct; ++i) {
    if (!std::isfinite(s->t_under[i]) || !std::isfinite(s->t_over[i]) || !std::isfinite(s->w_under[i]) ||
        !std::isfinite(s->w_over[i]) || s->w_under[i] < 0.f || s->w_over[i] < 0.f) {
      *err = "structure thresholds must be finite and weights finite and >= 0"; return DAO_E_ARG;
    }
  }
  if (opt->k_max < 1) { *err = "k_max must be >= 1"; return DAO_E_ARG; }
  if (opt->k_max > DAO_MAX_APERTURES) { *err = "k_max > DAO_MAX_APERTURES"; return DAO_E_UNSUPPORTED; }
  if (opt->master_max_iter < 0 || !(opt->master_tol >= 0.0) || !(opt->price_tol >= 0.0) ||
      (opt->master_method < 0 || opt->master_method > 3) || opt->sell_sigma < 0 ||
      !(opt->master_ls_tol > 0.0) || !(opt->master_ls_tol < 1.0) ||
      (opt->mlc_mode < DAO_MLC_CONSECUTIVE || opt->mlc_mode > DAO_MLC_CONNECTED)) {
    *err = "bad option value"; return DAO_E_ARG;
  }
  // MLC tables (host)
  if (mlc->beam_row_ptr[0] != 0 || mlc->beam_row_ptr[mlc->n_beams] != mlc->n_rows) {
    *err = "beam_row_ptr must start at 0 and end at n_rows"; return DAO_E_SHAPE;
  }
  int32_t max_rows = 0;
  for (int b = 0; b < mlc->n_beams; ++b) {
    const int32_t n = mlc->beam_row_ptr[b + 1] - mlc->beam_row_ptr[b];
    if (n < 0) { *err = "beam_row_ptr not monotone"; return DAO_E_SHAPE; }
    max_rows = std::max(max_rows, n);
  }
  if (mlc->row_bl_ptr[0] != 0 || mlc->row_bl_ptr[mlc->n_rows] != D->n_bl) {
    *err = "row_bl_ptr must start at 0 and end at n_bl"; return DAO_E_SHAPE;
  }
  for (int r = 0; r < mlc->n_rows; ++r)
    if (mlc->row_bl_ptr[r + 1] < mlc->row_bl_ptr[r]) { *err = "row_bl_ptr not monotone"; return DAO_E_SHAPE; }
  if (mlc->row_col0)
    for (int r = 0; r < mlc->n_rows; ++r)
      if (mlc->row_col0[r] < 0 || mlc->row_col0[r] > (1 << 20)) { *err = "row_col0 out of range"; return DAO_E_SHAPE; }
  dm->n_vox = D->n_vox; dm->n_bl = D->n_bl; dm->nnz = D->nnz;
  dm->n_beams = mlc->n_beams; dm->n_rows = mlc->n_rows; dm->k_max = opt->k_max;
  dm->max_rows = std::max(max_rows, 1);
  // the projected-Newton master handles pools up to kNewtonMaxK apertures; larger pools use method 1
  dm->master_method = (opt->master_method >= 2 && opt->k_max > kNewtonMaxK) ? 1 : opt->master_method;
  // the tcgen05 variant holds 8 block rows of the Hessian: beyond kNewtonTcMaxK apertures it is method 2, and says so
  // (dao_get_dims reports the method in effect)
  if (dm->master_method == 3 && opt->k_max > kNewtonTcMaxK) dm->master_method = 2;
  dm->n_struct = s->n_struct;
  dm->chain_states = 0;
  if (opt->mlc_mode == DAO_MLC_INTERDIGITATION || opt->mlc_mode == DAO_MLC_CONNECTED) {
    int32_t width = 0;
    for (int r = 0; r < mlc->n_rows; ++r)
      width = std::max(width, (mlc->row_col0 ? mlc->row_col0[r] : 0) + (mlc->row_bl_ptr[r + 1] - mlc->row_bl_ptr[r]));
    if (width > 1000) { *err = "interdigitation / connectedness pricing: beam wider than 1000 beamlets"; return DAO_E_UNSUPPORTED; }
    dm->chain_states = (width + 1) * (width + 1);
  }
  return DAO_OK;
}

static dao_status fetch_row_ptr(const dao_csr *D, std::vector<int32_t> *rp, std::string *err) {
  rp->resize((size_t)D->n_vox + 1);
  if (D->mem == DAO_MEM_HOST) {
    std::memcpy(rp->data(), D->row_ptr, rp->size() * sizeof(int32_t));
  } else {
    cudaError_t e = cudaMemcpy(rp->data(), D->row_ptr, rp->size() * sizeof(int32_t), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { *err = std::string("copy of row_ptr failed: ") + cudaGetErrorString(e); return DAO_E_CUDA; }
  }
  const std::vector<int32_t> &r = *rp;
  if (r[0] != 0 || (int64_t)r[D->n_vox] != D->nnz) { *err = "row_ptr[0] != 0 or row_ptr[n_vox] != nnz"; return DAO_E_SHAPE; }
  for (int32_t j = 0; j < D->n_vox; ++j)
    if (r[j + 1] < r[j]) { *err = "row_ptr not monotone"; return DAO_E_SHAPE; }
  return DAO_OK;
}

static int query_sm_count(int *device, std::string *err) {
  int dev = 0, n = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) { *err = std::string("no usable CUDA device: ") + cudaGetErrorString(e); return -1; }
  *device = dev;
  return n;
}

dao_status setup_sizes(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                       dao_sizes *out, std::string *err) {
  Dims dm{};
  dao_status st = check_args(D, mlc, s, opt, &dm, err);
  if (st != DAO_OK) return st;
  if (!out) { *err = "null output"; return DAO_E_ARG; }
  int dev = 0;
  const int n_sm = query_sm_count(&dev, err);
  if (n_sm < 0) return DAO_E_CUDA;
  std::vector<int32_t> rp;
  st = fetch_row_ptr(D, &rp, err);
  if (st != DAO_OK) return st;
  HostLayout L;
  const int sigma = effective_sigma(opt, D->n_vox);
  if (sigma >= D->n_vox && D->n_vox > 1) {
    // Sizes only: with ONE window sorted by descending length l_0 >= l_1 >= ..., slice s stores 32 l_{32 s} <= the sum of
    // the 32 lengths of slice s - 1, so the padded copy holds at most nnz + 32 l_0 elements -- no sort needed here
    // (dao_create computes the exact layout while the matrix uploads).
    int32_t max_len = 0;
    for (int32_t j = 0; j < D->n_vox; ++j) max_len = std::max(max_len, rp[j + 1] - rp[j]);
    L.n_vox_pad = (int32_t)align_up((size_t)std::max(D->n_vox, 1), 128);
    L.n_slices = L.n_vox_pad / kSellC;
    L.sell_elems = D->nnz + (int64_t)kSellC * max_len;
    if (L.sell_elems >= ((int64_t)1 << 32) - 64) { *err = "sliced-ELL copy of D would exceed 2^32 elements"; return DAO_E_UNSUPPORTED; }
  } else {
    st = make_layout(rp.data(), D->n_vox, sigma, &L, err);
    if (st != DAO_OK) return st;
  }
  Carver cw{nullptr};
  DevPtrs dp{};
  carve_workspace(cw, dm, L, &dp, n_sm);
  Carver cs{nullptr};
  ScratchPtrs sp{};
  carve_scratch(cs, dm, D->mem == DAO_MEM_HOST, &sp);
  out->workspace_bytes = align_up(cw.off, 256);
  out->scratch_bytes = align_up(cs.off, 256);
  return DAO_OK;
}

// ------------------------------------------------------------------------------------------
// setup kernels
// ------------------------------------------------------------------------------------------
enum { kErrColOrder = 1, kErrColRange = 2, kErrVal = 4, kErrStruct = 8 };

__global__ void k_validate(int32_t n_vox, int32_t n_bl, int32_t n_struct, const int32_t *__restrict__ row_ptr,
                           const int32_t *__restrict__ col, const float *__restrict__ val,
                           const int32_t *__restrict__ vs, int32_t *flags /* [0]=errors, [1..256]=struct counts */) {
  const int lane = threadIdx.x & 31;
  const int64_t warp_g = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  int err = 0;
  for (int64_t j = warp_g; j < n_vox; j += n_warps) {
    const int32_t lo = row_ptr[j], hi = row_ptr[j + 1];
    for (int32_t e = lo + lane; e < hi; e += 32) {
      const int32_t c = col[e];
      if (c < 0 || c >= n_bl) err |= kErrColRange;
      if (e > lo && col[e - 1] >= c) err |= kErrColOrder;
      const float v = val[e];
      if (!(v >= 0.f) || isinf(v)) err |= kErrVal;
    }
    if (lane == 0) {
      const int32_t s = vs[j];
      if (s < -1 || s >= n_struct) err |= kErrStruct;
      else if (s >= 0) atomicAdd(&flags[1 + s], 1);
    }
  }
  if (err) atomicOr(&flags[0], err);
}

__global__ void k_fill_sell(int32_t n_vox_pad, const int32_t *__restrict__ perm, const uint32_t *__restrict__ slice_off,
                            const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col,
                            const float *__restrict__ val, int32_t *__restrict__ sell_col,
                            float *__restrict__ sell_val) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_vox_pad) return;
  const int32_t slice = i / kSellC, r = i % kSellC;
  const uint32_t off = slice_off[slice];
  const int32_t slen = (int32_t)((slice_off[slice + 1] - off) / kSellC);
  const int32_t j = perm[i];
  int32_t lo = 0, n = 0;
  if (j >= 0) { lo = row_ptr[j]; n = row_ptr[j + 1] - lo; }
  for (int32_t k = 0; k < slen; ++k) {
    const size_t dst = (size_t)off + (size_t)k * kSellC + r;
    sell_col[dst] = k < n ? col[lo + k] : 0;
    sell_val[dst] = k < n ? val[lo + k] : 0.f;
  }
}

// per-voxel thresholds in the internal voxel order; flags non-finite values
__global__ void k_fill_vt(int32_t n_vox_pad, const int32_t *__restrict__ perm, const float *__restrict__ vt_in,
                          float *__restrict__ vt, int32_t *__restrict__ flags) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_vox_pad) return;
  const int32_t j = perm[i];
  const float t = j >= 0 ? vt_in[j] : 0.f;
  if (!isfinite(t)) atomicOr(flags, kErrVal);
  vt[i] = t;
}

__global__ void k_fill_sid(int32_t n_vox_pad, const int32_t *__restrict__ perm, const int32_t *__restrict__ vs,
                           uint8_t *__restrict__ sid) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_vox_pad) return;
  const int32_t j = perm[i];
  int32_t s = j >= 0 ? vs[j] : -1;
  sid[i] = (uint8_t)(s < 0 ? kNoStruct : s);
}

// expand D into (column key, voxel row, value) triples in CSR order (voxel ids are the caller's),
// and count the entries of every column (for t_ptr).
__global__ void k_expand(int32_t n_vox, const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col,
                         const float *__restrict__ val, int32_t *__restrict__ key, int32_t *__restrict__ row,
                         float *__restrict__ v, int32_t *__restrict__ col_count /* [n_bl+1], pre-zeroed */) {
  const int lane = threadIdx.x & 31;
  const int64_t warp_g = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t j = warp_g; j < n_vox; j += n_warps) {
    const int32_t lo = row_ptr[j], hi = row_ptr[j + 1];
    for (int32_t e = lo + lane; e < hi; e += 32) {
      const int32_t c = col[e];
      key[e] = c;
      row[e] = (int32_t)j;
      v[e] = val[e];
      atomicAdd(&col_count[c + 1], 1);
    }
  }
}

// in-place inclusive scan of n int32 by one CTA (setup only)
__global__ void __launch_bounds__(1024) k_scan_inclusive(int32_t *data, int64_t n) {
  __shared__ int32_t warp_tot[32];
  __shared__ int32_t carry_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (int64_t base = 0; base < n; base += 4096) {
    int32_t v[4];
    int32_t s = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t idx = base + (int64_t)tid * 4 + u;
      v[u] = idx < n ? data[idx] : 0;
      s += v[u];
    }
    int32_t inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      int32_t wt = warp_tot[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int32_t t = __shfl_up_sync(0xffffffffu, wt, o);
        if (lane >= o) wt += t;
      }
      warp_tot[lane] = wt;
    }
    __syncthreads();
    int32_t run = carry_s + (warp > 0 ? warp_tot[warp - 1] : 0) + (inc - s);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t idx = base + (int64_t)tid * 4 + u;
      run += v[u];
      if (idx < n) data[idx] = run;
    }
    __syncthreads();
    if (tid == 0) carry_s += warp_tot[31];
    __syncthreads();
  }
}

// Multi-CTA in-place inclusive scan (the radix sort's tile histograms: 256 x n_tiles counters, 3M on configs[1]; one
// CTA took 1.4 ms per pass): CTA b scans its chunk of kScanChunk elements and writes the chunk total, one CTA scans
// the totals (k_scan_inclusive), every chunk adds the total of the chunks before it.
__global__ void __launch_bounds__(1024) k_scan_chunks(int32_t *data, int64_t n, int32_t *sums) {
  __shared__ int32_t warp_tot[32];
  __shared__ int32_t carry_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t lo = (int64_t)blockIdx.x * kScanChunk, hi = lo + kScanChunk < n ? lo + kScanChunk : n;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (int64_t base = lo; base < hi; base += 4096) {
    int32_t v[4];
    int32_t sm = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t idx = base + (int64_t)tid * 4 + u;
      v[u] = idx < hi ? data[idx] : 0;
      sm += v[u];
    }
    int32_t inc = sm;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      int32_t wt = warp_tot[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int32_t t = __shfl_up_sync(0xffffffffu, wt, o);
        if (lane >= o) wt += t;
      }
      warp_tot[lane] = wt;
    }
    __syncthreads();
    int32_t run = carry_s + (warp > 0 ? warp_tot[warp - 1] : 0) + (inc - sm);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t idx = base + (int64_t)tid * 4 + u;
      run += v[u];
      if (idx < hi) data[idx] = run;
    }
    __syncthreads();
    if (tid == 1023) carry_s = run;
    __syncthreads();
  }
  if (tid == 0) sums[blockIdx.x] = carry_s;
}
__global__ void __launch_bounds__(1024) k_scan_add(int32_t *data, int64_t n, const int32_t *__restrict__ sums) {
  if (blockIdx.x == 0) return;
  const int32_t add = sums[blockIdx.x - 1];
  const int64_t lo = (int64_t)blockIdx.x * kScanChunk, hi = lo + kScanChunk < n ? lo + kScanChunk : n;
  for (int64_t i = lo + threadIdx.x; i < hi; i += 1024) data[i] += add;
}

// LSD radix pass, 8 bits: (1) per-tile digit histogram, (2) scan of [digit][tile] counts,
// (3) stable scatter.  Elements are taken warp-blocked (warp w of a tile owns 32*kRadixItems
// consecutive elements, visited 32 at a time), so index order = visiting order.
__global__ void __launch_bounds__(kRadixThreads) k_radix_hist(const int32_t *__restrict__ key, int64_t n, int shift,
                                                             int32_t n_tiles, int32_t *__restrict__ tile_hist) {
  __shared__ int32_t hist[256];
  hist[threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t base = (int64_t)blockIdx.x * kRadixTile + (int64_t)warp * 32 * kRadixItems;
#pragma unroll
  for (int r = 0; r < kRadixItems; ++r) {
    const int64_t idx = base + r * 32 + lane;
    if (idx < n) atomicAdd(&hist[(key[idx] >> shift) & 255], 1);
  }
  __syncthreads();
  tile_hist[(size_t)threadIdx.x * n_tiles + blockIdx.x] = hist[threadIdx.x];
}

__global__ void __launch_bounds__(kRadixThreads) k_radix_scatter(
    const int32_t *__restrict__ key, const int32_t *__restrict__ row, const float *__restrict__ val, int64_t n,
    int shift, int32_t n_tiles, const int32_t *__restrict__ tile_scan /* inclusive scan of tile_hist */,
    int32_t *__restrict__ okey, int32_t *__restrict__ orow, float *__restrict__ oval) {
  __shared__ int32_t cnt[kRadixThreads / 32][256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < (kRadixThreads / 32) * 256; i += kRadixThreads) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kRadixTile + (int64_t)warp * 32 * kRadixItems;
  int32_t k[kRadixItems], rk[kRadixItems];
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int r = 0; r < kRadixItems; ++r) {
    const int64_t idx = base + r * 32 + lane;
    const bool valid = idx < n;
    k[r] = valid ? key[idx] : 0;
    const int d = valid ? ((k[r] >> shift) & 255) : (256 + lane);   // invalid lanes match nobody
    const unsigned m = __match_any_sync(0xffffffffu, d);
    const int leader = __ffs(m) - 1;
    int32_t prev = 0;
    if (valid && lane == leader) {
      prev = cnt[warp][d];
      cnt[warp][d] = prev + __popc(m);
    }
    prev = __shfl_sync(0xffffffffu, prev, leader);
    rk[r] = prev + __popc(m & lt);
    __syncwarp();
  }
  __syncthreads();
  {
    // exclusive offsets: global start of (digit, tile) + counts of the preceding warps
    const int d = threadIdx.x;
    const size_t pos = (size_t)d * n_tiles + blockIdx.x;
    int32_t run = pos > 0 ? tile_scan[pos - 1] : 0;
#pragma unroll
    for (int w = 0; w < kRadixThreads / 32; ++w) {
      const int32_t t = cnt[w][d];
      cnt[w][d] = run;
      run += t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kRadixItems; ++r) {
    const int64_t idx = base + r * 32 + lane;
    if (idx < n) {
      const int d = (k[r] >> shift) & 255;
      const int32_t dst = cnt[warp][d] + rk[r];
      okey[dst] = k[r];
      orow[dst] = row[idx];
      oval[dst] = val[idx];
    }
  }
}

__global__ void k_fill_i32(int32_t *p, int64_t n, int32_t v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}


// ------------------------------------------------------------------------------------------
// dao_create body
// ------------------------------------------------------------------------------------------
#define SETUP_CUDA(call)                                                                  \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                        \
      return DAO_E_CUDA;                                                                  \
    }                                                                                     \
  } while (0)

static int grid_for(int64_t n, int threads, int cap = 1 << 20) {
  int64_t g = (n + threads - 1) / threads;
  if (g < 1) g = 1;
  if (g > cap) g = cap;
  return (int)g;
}

dao_status setup_build(Ctx *c, const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, void *workspace,
                       size_t workspace_bytes, void *scratch, size_t scratch_bytes) {
  Dims dm{};
  dao_status st = check_args(D, mlc, s, &c->opt, &dm, &c->err);
  if (st != DAO_OK) return st;
  c->opt.master_method = dm.master_method;
  c->n_sm = query_sm_count(&c->device, &c->err);
  if (c->n_sm < 0) return DAO_E_CUDA;
  if (!workspace || !scratch || ((uintptr_t)workspace & 255) || ((uintptr_t)scratch & 255)) {
    c->err = "workspace and scratch must be non-null and 256-byte aligned";
    return DAO_E_ALLOC;
  }
  std::vector<int32_t> rp;
  st = fetch_row_ptr(D, &rp, &c->err);
  if (st != DAO_OK) return st;
  Carver cs{reinterpret_cast<unsigned char *>(scratch)};
  ScratchPtrs sp{};
  const bool host_in = D->mem == DAO_MEM_HOST;
  carve_scratch(cs, dm, host_in, &sp);
  if (cs.off > scratch_bytes) {
    c->err = "workspace or scratch smaller than dao_workspace_bytes reported";
    return DAO_E_ALLOC;
  }
  // the large uploads go out first: the host computes the sliced-ELL layout (a sort of the rows by length) while
  // they are in flight
  if (host_in) {
    SETUP_CUDA(cudaMemcpyAsync(sp.row_ptr, D->row_ptr, ((size_t)dm.n_vox + 1) * 4, cudaMemcpyHostToDevice, c->stream));
    if (dm.nnz > 0) {
      SETUP_CUDA(cudaMemcpyAsync(sp.col, D->col_idx, (size_t)dm.nnz * 4, cudaMemcpyHostToDevice, c->stream));
      SETUP_CUDA(cudaMemcpyAsync(sp.val, D->val, (size_t)dm.nnz * 4, cudaMemcpyHostToDevice, c->stream));
    }
    SETUP_CUDA(cudaMemcpyAsync(sp.vs, s->vox_struct, (size_t)dm.n_vox * 4, cudaMemcpyHostToDevice, c->stream));
  }
  HostLayout L;
  c->opt.sell_sigma = effective_sigma(&c->opt, D->n_vox);
  st = make_layout(rp.data(), D->n_vox, c->opt.sell_sigma, &L, &c->err);
  if (st != DAO_OK) return st;

  Carver cw{reinterpret_cast<unsigned char *>(workspace)};
  carve_workspace(cw, dm, L, &c->d, c->n_sm);
  if (cw.off > workspace_bytes) {
    c->err = "workspace or scratch smaller than dao_workspace_bytes reported";
    return DAO_E_ALLOC;
  }
  c->n_vox = dm.n_vox; c->n_bl = dm.n_bl; c->nnz = dm.nnz;
  c->n_beams = dm.n_beams; c->n_rows = dm.n_rows; c->n_struct = s->n_struct;
  c->n_vox_pad = L.n_vox_pad; c->n_slices = L.n_slices; c->sell_elems = L.sell_elems;
  c->max_rows_per_beam = dm.max_rows;
  c->beam_row_ptr.assign(mlc->beam_row_ptr, mlc->beam_row_ptr + dm.n_beams + 1);
  c->row_bl_ptr.assign(mlc->row_bl_ptr, mlc->row_bl_ptr + dm.n_rows + 1);
  c->row_col0.assign((size_t)dm.n_rows, 0);
  if (mlc->row_col0) c->row_col0.assign(mlc->row_col0, mlc->row_col0 + dm.n_rows);
  c->max_beam_width = 0;
  c->max_row_len = 0;
  for (int r = 0; r < dm.n_rows; ++r) c->max_row_len = std::max(c->max_row_len, c->row_bl_ptr[r + 1] - c->row_bl_ptr[r]);
  for (int r = 0; r < dm.n_rows; ++r)
    c->max_beam_width = std::max(c->max_beam_width, c->row_col0[r] + (c->row_bl_ptr[r + 1] - c->row_bl_ptr[r]));
  if (c->opt.mlc_mode == DAO_MLC_JAWS_ONLY &&
      (size_t)dm.max_rows * (size_t)(c->max_beam_width + 1) * sizeof(double) > (size_t)200 * 1024) {
    c->err = "jaws-only pricing: rows x lateral width of a beam exceeds the shared-memory table (200 KB)";
    return DAO_E_UNSUPPORTED;
  }
  if ((c->opt.mlc_mode == DAO_MLC_INTERDIGITATION || c->opt.mlc_mode == DAO_MLC_CONNECTED) &&
      (chain_pricing_smem(dm.max_rows, c->max_beam_width) > (size_t)200 * 1024 || c->max_beam_width > 30000)) {
    c->err = "interdigitation / connectedness pricing: rows x leaf states of a beam exceed the shared-memory tables (200 KB)";
    return DAO_E_UNSUPPORTED;
  }
  cudaStream_t q = c->stream;
  DevPtrs &d = c->d;

  // ---- inputs on the device ----
  const int32_t *d_row_ptr, *d_col, *d_vs;
  const float *d_val;
  if (host_in) {                 // uploaded above, before the host computed the layout
    d_row_ptr = sp.row_ptr; d_col = sp.col; d_val = sp.val; d_vs = sp.vs;
  } else {
    d_row_ptr = D->row_ptr; d_col = D->col_idx; d_val = D->val; d_vs = s->vox_struct;
  }

  // ---- validate + structure sizes ----
  SETUP_CUDA(cudaMemsetAsync(sp.flags, 0, 260 * sizeof(int32_t), q));
  k_validate<<<grid_for((int64_t)dm.n_vox * 32, 256, c->n_sm * 16), 256, 0, q>>>(dm.n_vox, dm.n_bl, s->n_struct, d_row_ptr,
                                                                             d_col, d_val, d_vs, sp.flags);
  SETUP_CUDA(cudaGetLastError());
  int32_t h_flags[260];
  SETUP_CUDA(cudaMemcpyAsync(h_flags, sp.flags, sizeof(h_flags), cudaMemcpyDeviceToHost, q));
  SETUP_CUDA(cudaStreamSynchronize(q));
  if (h_flags[0] & kErrColRange) { c->err = "col_idx out of range"; return DAO_E_SHAPE; }
  if (h_flags[0] & kErrColOrder) { c->err = "col_idx not strictly ascending inside a row"; return DAO_E_SHAPE; }
  if (h_flags[0] & kErrStruct) { c->err = "vox_struct out of range"; return DAO_E_SHAPE; }
  if (h_flags[0] & kErrVal) { c->err = "val must be finite and >= 0"; return DAO_E_ARG; }

  // per-structure penalty table, eq. (9)-(10): alpha_s/|v_s|, beta_s/|v_s|, T_s^-, T_s^+
  {
    std::vector<StructEntry> tab(256, StructEntry{0.0, 0.0, 0.0, 0.0});
    for (int i = 0; i < s->n_struct; ++i) {
      // |v_s|: the context's own count, or the caller's count over the whole problem (voxel-row slab)
      const double n = s->struct_count ? (double)s->struct_count[i] : (double)h_flags[1 + i];
      const double div = s->per_voxel_weights ? 1.0 : n;       // eq. 3-4 as given, or eq. 9-10 per |v_s|
      tab[i].a = n > 0 ? (double)s->w_under[i] / div : 0.0;
      tab[i].b = n > 0 ? (double)s->w_over[i] / div : 0.0;
      tab[i].tm = (double)s->t_under[i];
      tab[i].tp = (double)s->t_over[i];
    }
    SETUP_CUDA(cudaMemcpyAsync(d.stab, tab.data(), 256 * sizeof(StructEntry), cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaStreamSynchronize(q));
  }

  // ---- layout tables ----
  SETUP_CUDA(cudaMemcpyAsync(d.perm, L.perm.data(), (size_t)L.n_vox_pad * 4, cudaMemcpyHostToDevice, q));
  SETUP_CUDA(cudaMemcpyAsync(d.inv_perm, L.inv_perm.data(), (size_t)dm.n_vox * 4, cudaMemcpyHostToDevice, q));
  SETUP_CUDA(cudaMemcpyAsync(d.slice_off, L.slice_off.data(), ((size_t)L.n_slices + 1) * 4, cudaMemcpyHostToDevice, q));
  k_fill_sell<<<grid_for(L.n_vox_pad, 128), 128, 0, q>>>(L.n_vox_pad, d.perm, d.slice_off, d_row_ptr, d_col, d_val,
                                                        d.sell_col, d.sell_val);
  SETUP_CUDA(cudaGetLastError());
  k_fill_sid<<<grid_for(L.n_vox_pad, 256), 256, 0, q>>>(L.n_vox_pad, d.perm, d_vs, d.sid);
  SETUP_CUDA(cudaGetLastError());
  c->has_vt = s->vox_threshold != nullptr;
  if (c->has_vt) {
    const float *d_vt = s->vox_threshold;
    if (host_in) {
      SETUP_CUDA(cudaMemcpyAsync(sp.vt, s->vox_threshold, (size_t)dm.n_vox * 4, cudaMemcpyHostToDevice, q));
      d_vt = sp.vt;
    }
    SETUP_CUDA(cudaMemsetAsync(sp.flags, 0, sizeof(int32_t), q));
    k_fill_vt<<<grid_for(L.n_vox_pad, 256), 256, 0, q>>>(L.n_vox_pad, d.perm, d_vt, d.vt, sp.flags);
    SETUP_CUDA(cudaGetLastError());
    int32_t f = 0;
    SETUP_CUDA(cudaMemcpyAsync(&f, sp.flags, sizeof(f), cudaMemcpyDeviceToHost, q));
    SETUP_CUDA(cudaStreamSynchronize(q));
    if (f & kErrVal) { c->err = "vox_threshold must be finite"; return DAO_E_ARG; }
  } else {
    SETUP_CUDA(cudaMemsetAsync(d.vt, 0, (size_t)L.n_vox_pad * 4, q));
  }

  // ---- CSR of D^T: expand, count columns, stable radix sort on the column index ----
  const int64_t ntc = tchunks_of(dm.nnz);
  c->n_tchunks = (int32_t)ntc;
  SETUP_CUDA(cudaMemsetAsync(d.t_ptr, 0, ((size_t)dm.n_bl + 2) * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.t_row, 0, ((size_t)ntc * kTChunk + 64) * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.t_val, 0, ((size_t)ntc * kTChunk + 64) * 4, q));
  std::vector<int32_t> h_tptr((size_t)dm.n_bl + 1, 0);
  if (dm.nnz > 0) {
    k_expand<<<grid_for((int64_t)dm.n_vox * 32, 256, c->n_sm * 16), 256, 0, q>>>(dm.n_vox, d_row_ptr, d_col, d_val, sp.keyA,
                                                                             sp.rowA, sp.valA, d.t_ptr);
    SETUP_CUDA(cudaGetLastError());
    k_scan_inclusive<<<1, 1024, 0, q>>>(d.t_ptr, (int64_t)dm.n_bl + 1);
    SETUP_CUDA(cudaGetLastError());
    int bits = 1;
    while (((int64_t)1 << bits) < (int64_t)dm.n_bl) ++bits;
    const int n_pass = (bits + 7) / 8;
    const int32_t n_tiles = (int32_t)((dm.nnz + kRadixTile - 1) / kRadixTile);
    int32_t *ik = sp.keyA, *ir = sp.rowA, *ok = sp.keyB, *orow = sp.rowB;
    float *iv = sp.valA, *ov = sp.valB;
    for (int pass = 0; pass < n_pass; ++pass) {
      const bool last = pass == n_pass - 1;
      int32_t *dst_row = last ? d.t_row : orow;
      float *dst_val = last ? d.t_val : ov;
      k_radix_hist<<<n_tiles, kRadixThreads, 0, q>>>(ik, dm.nnz, pass * 8, n_tiles, sp.tile_hist);
      SETUP_CUDA(cudaGetLastError());
      {
        const int64_t n_scan = (int64_t)256 * n_tiles;
        const int n_chunks = (int)((n_scan + kScanChunk - 1) / kScanChunk);
        k_scan_chunks<<<n_chunks, 1024, 0, q>>>(sp.tile_hist, n_scan, sp.scan_sums);
        k_scan_inclusive<<<1, 1024, 0, q>>>(sp.scan_sums, (int64_t)n_chunks);
        k_scan_add<<<n_chunks, 1024, 0, q>>>(sp.tile_hist, n_scan, sp.scan_sums);
      }
      SETUP_CUDA(cudaGetLastError());
      k_radix_scatter<<<n_tiles, kRadixThreads, 0, q>>>(ik, ir, iv, dm.nnz, pass * 8, n_tiles, sp.tile_hist, ok, dst_row,
                                                       dst_val);
      SETUP_CUDA(cudaGetLastError());
      std::swap(ik, ok); std::swap(ir, orow); std::swap(iv, ov);
    }
    SETUP_CUDA(cudaMemcpyAsync(h_tptr.data(), d.t_ptr, ((size_t)dm.n_bl + 1) * 4, cudaMemcpyDeviceToHost, q));
    SETUP_CUDA(cudaStreamSynchronize(q));
    if ((int64_t)h_tptr[dm.n_bl] != dm.nnz) { c->err = "internal error: transposed pointer mismatch"; return DAO_E_CUDA; }
  }
  // chunk tables of the transposed SpMV
  {
    std::vector<int32_t> first((size_t)ntc + 1, 0), segbase((size_t)ntc + 2, 0);
    int32_t row = 0;
    int64_t total = 0;
    for (int64_t ch = 0; ch < ntc; ++ch) {
      const int64_t cbeg = ch * kTChunk, cend = std::min<int64_t>(cbeg + kTChunk, dm.nnz);
      while (h_tptr[row + 1] <= cbeg) ++row;            // row containing element cbeg
      int32_t lastrow = row;
      while (h_tptr[lastrow + 1] < cend) ++lastrow;     // row containing element cend-1
      first[ch] = row;
      segbase[ch] = (int32_t)total;
      total += lastrow - row + 1;
    }
    segbase[ntc] = (int32_t)total;
    c->n_tsegs = (int32_t)total;
    if ((size_t)total > (size_t)ntc + (size_t)dm.n_bl + 2) { c->err = "internal error: segment count"; return DAO_E_CUDA; }
    SETUP_CUDA(cudaMemcpyAsync(d.t_first_row, first.data(), ((size_t)ntc + 1) * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaMemcpyAsync(d.t_seg_base, segbase.data(), ((size_t)ntc + 2) * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaStreamSynchronize(q));
  }

  // ---- MLC lookup tables ----
  {
    std::vector<int32_t> bl_row((size_t)dm.n_bl), row_beam((size_t)dm.n_rows);
    for (int b = 0; b < dm.n_beams; ++b)
      for (int r = c->beam_row_ptr[b]; r < c->beam_row_ptr[b + 1]; ++r) row_beam[r] = b;
    for (int r = 0; r < dm.n_rows; ++r)
      for (int i = c->row_bl_ptr[r]; i < c->row_bl_ptr[r + 1]; ++i) bl_row[i] = r;
    SETUP_CUDA(cudaMemcpyAsync(d.beam_row_ptr, c->beam_row_ptr.data(), ((size_t)dm.n_beams + 1) * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaMemcpyAsync(d.row_bl_ptr, c->row_bl_ptr.data(), ((size_t)dm.n_rows + 1) * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaMemcpyAsync(d.bl_row, bl_row.data(), (size_t)dm.n_bl * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaMemcpyAsync(d.row_beam, row_beam.data(), (size_t)dm.n_rows * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaMemcpyAsync(d.row_col0, c->row_col0.data(), (size_t)dm.n_rows * 4, cudaMemcpyHostToDevice, q));
    SETUP_CUDA(cudaStreamSynchronize(q));
  }

  // ---- zero the state ----
  const size_t vp = (size_t)L.n_vox_pad;
  SETUP_CUDA(cudaMemsetAsync(d.state, 0, sizeof(DevState), q));
  SETUP_CUDA(cudaMemsetAsync(d.fmo_state, 0, sizeof(FmoState), q));
  SETUP_CUDA(cudaMemsetAsync(d.x, 0, (size_t)dm.n_bl * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.xmask, 0, (size_t)dm.n_bl * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.z, 0, vp * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.g, 0, vp * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.w, 0, (size_t)dm.n_bl * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.y, 0, DAO_MAX_APERTURES * 8, q));
  SETUP_CUDA(cudaMemsetAsync(d.mdz, 0, vp * 8, q));
  c->nwt = layout_of_master(dm, L.n_vox_pad);
  c->red_stride = c->nwt.T ? c->nwt.n_red : kMaxRedux;
  SETUP_CUDA(cudaMemsetAsync(d.mz, 0, (c->nwt.T ? (size_t)c->nwt.n_tiles * (size_t)c->nwt.T : vp) * 8, q));
  {
    const size_t g = (size_t)std::min(c->n_sm * kMasterCtasPerSm, kMasterMaxGrid);
    SETUP_CUDA(cudaMemsetAsync(d.ll_part, 0, 2 * g * (size_t)c->red_stride * sizeof(uint4), q));
    SETUP_CUDA(cudaMemsetAsync(d.ll_result, 0, 2 * (size_t)c->red_stride * sizeof(uint4), q));
  }
  // the tiled dose block is read with its padding (tile tails, the 4 pad floats of every column): finite zeros
  if (c->nwt.T) SETUP_CUDA(cudaMemsetAsync(d.A, 0, (size_t)c->nwt.n_tiles * (size_t)c->nwt.tile_stride * 4, q));
  SETUP_CUDA(newton_fill_tile_meta(c));
  SETUP_CUDA(cudaMemsetAsync(d.m_epoch, 0, 64 * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.m_prof, 0, kMasterProfSlots * 8, q));
  SETUP_CUDA(cudaMemsetAsync(d.ap_beam, 0, (size_t)dm.k_max * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.ap_hash, 0, (size_t)dm.k_max * 8, q));
  SETUP_CUDA(cudaMemsetAsync(d.ap_left, 0, (size_t)dm.k_max * dm.max_rows * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.ap_right, 0, (size_t)dm.k_max * dm.max_rows * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.history, 0, (size_t)dm.k_max * sizeof(dao_iter_record), q));
  SETUP_CUDA(cudaMemsetAsync(d.left, 0, (size_t)dm.n_rows * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.right, 0, (size_t)dm.n_rows * 4, q));
  SETUP_CUDA(cudaMemsetAsync(d.vstar, 0, (size_t)dm.n_rows * 8, q));
  SETUP_CUDA(cudaMemsetAsync(d.beam_price, 0, (size_t)dm.n_beams * 8, q));

  spmv_configure(c);
  SETUP_CUDA(master_configure(c));
  SETUP_CUDA(cudaStreamSynchronize(q));
  return DAO_OK;
}

}  // namespace dao
