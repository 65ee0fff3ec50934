// dao_internal.cuh -- shared declarations of the CUDA library behind include/dao.h.
// Nothing here is shared with oracle/ (the fp64 CPU oracle is independent test infrastructure).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "dao.h"

namespace dao {

// ------------------------------------------------------------------------------------------
// Tunables (compile time)
// ------------------------------------------------------------------------------------------
constexpr int kSellC = 32;             // rows per sliced-ELL slice: one warp, lane = row
constexpr int kSpmvThreads = 512;      // CTA size of the direct-load SELL SpMV kernel
constexpr int kSpmvRingThreads = 512;  // max CTA size of the TMA-ring SELL SpMV kernel (one CTA per SM)
constexpr int kSpmvXSmemMax = 24576;   // x is staged in shared memory when n_bl <= this (96 KB fp32)
constexpr int kTChunk = 4096;          // elements of D^T per CTA in the transposed SpMV
constexpr int kTThreads = 256;
constexpr int kTCtasPerSm = 6;         // persistent CTAs per SM of the transposed SpMV
constexpr int kMasterWorkers = 512;    // worker threads of the persistent master kernel (one CTA per SM)
constexpr int kMasterThreads = kMasterWorkers + 32;   // + the producer warp that streams A through the ring
#ifndef DAO_MASTER_CTAS_PER_SM
#define DAO_MASTER_CTAS_PER_SM 1
#endif
constexpr int kMasterCtasPerSm = DAO_MASTER_CTAS_PER_SM;   // resident CTAs of the master per SM.  2 (34 warps per SM, one strip per warp) was measured on cfg1: the passes
                                       // take the same time (L2-side limit, not warp latency) and the grid reductions over 296 CTAs double: slower
constexpr int kMasterStrips = kMasterCtasPerSm == 1 ? 2 : 1;   // 128-voxel strips per worker warp and stage
constexpr int kMasterTileVox = 16 * 128 * kMasterStrips;   // voxels per ring stage: 16 worker warps x strips x 128
constexpr int kMasterColBytes = kMasterTileVox * 4;      // one column of one tile
#ifndef DAO_MASTER_COLS_PER_STAGE
#define DAO_MASTER_COLS_PER_STAGE 2
#endif
constexpr int kMasterColsPerStage = DAO_MASTER_COLS_PER_STAGE;   // a ring stage holds this many consecutive columns (even)
                                                        // behind ONE full/empty mbarrier pair: the barrier traffic per byte,
                                                        // not the memory system, limits the passes (measured: 1 -> 2 columns
                                                        // per stage made them 16 % faster)
constexpr int kMasterStageBytes = kMasterColsPerStage * kMasterColBytes;
constexpr int kMasterMaxStages = 10 / kMasterColsPerStage + 1;
constexpr int kMasterMaxGrid = 160 * kMasterCtasPerSm;    // CTAs of the master kernel (capped)
constexpr int kMasterProfSlots = 16;   // phase timers of the master (ns): 0 init, 1 G pass, 2 G reduce, 3 direction,
                                       // 4 D pass, 5 D reduce, 6 line search; 7 line-search evaluations,
                                       // 8 iterations, 9 calls, 10 publish
constexpr int kFmoLsGridMax = 1024;   // CTAs of the FMO line-search kernels
constexpr int kMaxStruct = 255;
constexpr int kNoStruct = 255;         // sid value of a voxel without penalty
constexpr int kMaxRedux = DAO_MAX_APERTURES + 8;   // doubles per grid reduction in the master (methods 0, 1)

// ---- master_method = 2, 3 (projected Newton, dao_newton.cu) ----
constexpr int kNewtonTcMaxK = 56;  // largest pool method 3 handles (8 block rows of the augmented Hessian = the 64 rows of one operand half); larger k_max: method 2
constexpr int kNewtonMaxK = 103;   // largest pool methods 2, 3 handle (13 block rows of the Hessian); larger k_max: method 1
// The aperture-dose block is stored TILED: tile t holds T voxels (voxel i sits in tile i mod n_tiles at slot
// i / n_tiles, a_index) as rows of TP = T + 4 floats: `meta_rows` rows with the structure ids and per-voxel
// thresholds of its voxels, then its k_max columns back to back, so that the meta rows and the K live columns of
// a tile are ONE contiguous range = one bulk copy.
struct NewtonLayout {
  int32_t T = 0;            // voxels per tile (0: plain aperture-major layout, methods 0 and 1)
  int32_t TP = 0;           // floats per column inside a tile
  int32_t n_tiles = 0;      // ceil(n_vox_pad / T)
  int64_t tile_stride = 0;  // floats between consecutive tiles = (meta_rows + k_max) * TP
  int32_t n_stages = 0;     // ring stages of stage_bytes
  int32_t stage_bytes = 0;  // k_max * TP * 4 rounded to 128
  int32_t nb_max = 0;       // 8x8 block rows of the augmented Hessian at K = k_max: ceil((k_max + 1) / 8)
  int32_t n_red = 0;        // doubles per grid reduction: nb_max (nb_max + 1) / 2 * 64 + 8
  int32_t AC = 0;           // active voxels per chunk of the Hessian phase
  int32_t lbuf_doubles = 0; // shared buffer of the LDL^T factorisation and of the fp64 tile W of the Hessian phase
  size_t smem = 0;          // dynamic shared memory of k_master_newton
  // master_method = 3: the Hessian on the 5th-generation tensor cores (tcgen05, TF32 hi/lo split, TMEM accumulators)
  int32_t tc = 0;           // 1: k_master_newton<true>
  int32_t kp = 0;           // rows of one half (hi or lo) of the operand tile: 64 (method 3 exists for k_max <= kNewtonTcMaxK = 56 only)
  int32_t lbo = 0;          // bytes between the two 16-byte K-halves of an MMA k-step (core matrices adjacent along the voxels)
  int32_t sbo = 0;          // bytes between groups of 8 operand rows
  int32_t w_bytes = 0;      // bytes of one operand tile: (2 kp / 8) sbo
  int32_t tmem_cols = 0;    // TMEM columns allocated per CTA (power of two >= 32)
  int32_t meta_rows = 0;    // rows of TP floats at the head of every tile (structure ids, thresholds) before column 0
};

// ------------------------------------------------------------------------------------------
// Device-resident state shared by the kernels of one context (one instance in global memory).
// The host reads it once per column-generation iteration.
// ------------------------------------------------------------------------------------------
struct DevState {
  // pool
  int32_t K;               // apertures in the pool
  int32_t done;            // 1: pricing proved optimality; 2: stalled on a duplicate candidate after an unconverged master
  // pending candidate (result of the last pricing)
  int32_t cand_valid;
  int32_t cand_beam;
  int32_t cand_dup;
  int32_t cand_nopen;
  double cand_price;
  double w_abs_max;
  // last dose evaluation
  double F;
  // last master solve
  int32_t m_iters;
  int32_t m_hit_max;
  int32_t m_restarts;
  int32_t m_added;         // 1: the master appended the candidate
  double m_F;
  double m_kkt;
  double m_pg;
  // counters used by last-block reductions (self-resetting)
  uint32_t ticket_spmv;
  uint32_t ticket_misc;
  // grid barrier of the master kernel
  uint32_t bar_count;
  uint32_t bar_gen;
  int64_t pg_iter_total;
  int64_t pass_total;      // passes over the aperture-dose block A (each reads 4 V K bytes) since dao_create / dao_reset
  int32_t m_passes;        // passes over A of the last master solve
  int32_t n_hit_max;       // master solves that stopped on the iteration cap since dao_create / dao_reset
  int32_t n_duplicates;
  unsigned long long cand_hash;   // aperture_hash of the pending candidate
  int32_t price_maxlen;    // longest leaf row of caller-provided MLC tables (dao_price_from_w), decided on the device
};

// Device state of the FMO solve (dao_fmo.cu); the host reads it every few iterations.
struct FmoState {
  double F;                // objective at the current x
  double slope0;           // phi'(0) = p . w
  double tmax;             // largest feasible step along p
  double t;                // current trial / accepted step
  double lo, slo, hi, shi; // bracket of the root of phi' (hi = inf: none yet)
  double c1, c2;           // phi'(t), phi''(t) of the last evaluation
  double pg_max, kkt, x_max;
  double F_prev;           // objective of the previous iteration (stall detection)
  double t_est;            // bending horizon of the next direction (2 x the last accepted step; 0: none)
  int32_t done;            // 1: converged or iteration cap; every FMO kernel returns at once
  int32_t converged;
  int32_t hit_max;
  int32_t iters;
  int32_t ls_done;         // 1: the step t is accepted
  int32_t at_bound;        // accepted step ends on the bound of variable ib
  int32_t ib;
  int32_t force_restart;
  int32_t since_restart;
  int32_t restarts;
  int32_t ls_evals;
  int32_t stall;           // consecutive iterations without a decrease of F beyond fp64 rounding
  uint32_t ticket;
};

struct StructEntry {       // per-structure penalty parameters of eq. (9)-(10), already divided by |v_s|
  double a;                // alpha_s / |v_s|
  double b;                // beta_s  / |v_s|
  double tm;               // T_s^-
  double tp;               // T_s^+
};

// All device pointers of a context.  Voxel-space arrays are in the INTERNAL voxel order
// (internal row i holds the caller's voxel perm[i]) EXCEPT z and g, which the dose SpMV scatters
// straight into the caller's order (D^T gathers g by caller voxel id, where a beamlet's voxels
// form contiguous runs).
struct DevPtrs {
  // sliced ELL of D
  int32_t *sell_col;
  float *sell_val;
  uint32_t *slice_off;     // [n_slices+1] element offsets
  int32_t *perm;           // [n_vox_pad] internal -> caller voxel (-1 for padding rows)
  int32_t *inv_perm;       // [n_vox]     caller voxel -> internal
  uint8_t *sid;            // [n_vox_pad] structure id or kNoStruct
  StructEntry *stab;       // [256]
  float *vt;               // [n_vox_pad] per-voxel threshold T_j (re-optimisation mode), internal order
  // CSR of D^T (rows = beamlets, entries = the CALLER's voxel ids: pi is kept in the caller's order)
  int32_t *t_ptr;          // [n_bl+1]
  int32_t *t_row;          // [nnz padded to kTChunk] caller voxel ids, ascending inside a row
  float *t_val;
  int32_t *t_first_row;    // [n_tchunks]
  int32_t *t_seg_base;     // [n_tchunks+1]
  double *t_segsum;        // [n_tsegs]
  // MLC tables
  int32_t *beam_row_ptr;   // [n_beams+1]
  int32_t *row_bl_ptr;     // [n_rows+1]
  int32_t *bl_row;         // [n_bl]
  int32_t *row_beam;       // [n_rows]
  int32_t *row_col0;       // [n_rows] lateral position of the first beamlet of every row
  int32_t *chain_from;     // [n_rows][(W+1)^2] back-pointers of the chain pricing modes (W = widest beam)
  // vectors
  float *x;                // [n_bl]
  float *xmask;            // [n_bl]
  float *z;                // [n_vox_pad] caller order
  float *g;                // [n_vox_pad] caller order
  float *w;                // [n_bl]
  double *f_part;          // [grid of the spmv kernel]
  // pricing
  double *vstar;           // [n_rows]
  int32_t *left, *right;   // [n_rows]
  double *row_absmax;      // [n_rows]
  double *beam_price;      // [n_beams]
  double *beam_absmax;     // [n_beams]
  // pool
  int32_t *ap_beam;        // [k_max]
  unsigned long long *ap_hash;   // [k_max] aperture_hash of every pool aperture (duplicate test: compare, then verify)
  int32_t *ap_left;        // [k_max * max_rows_per_beam]
  int32_t *ap_right;
  float *A;                // dose block: [k_max][n_vox_pad] aperture-major (methods 0, 1) or tiled (methods 2, 3: NewtonLayout, a_index)
  double *y;               // [k_max]
  // master
  double *mz;              // z = A y: [n_vox_pad] internal order (methods 0, 1) or [n_tiles * T] in the tiled order (methods 2, 3)
  double *mdz;             // [n_vox_pad] dz = A p
  uint4 *ll_part;          // [2][n_cta][kMaxRedux] flagged slots {lo32, epoch, hi32, epoch} of the grid reductions
  uint4 *ll_result;        // [2][kMaxRedux]
  uint32_t *m_epoch;       // reduction epoch (monotone over the life of the context)
  unsigned long long *m_prof;  // [kMasterProfSlots]
  // FMO workload
  float *fmo_p;            // [n_bl] search direction (fp32 values: x += t p and dz = D p stay consistent)
  float *fmo_pgold;        // [n_bl] previous projected steepest-descent direction
  float *fmo_dz;           // [n_vox_pad] dz = D p, internal order
  double *fmo_part;        // [2 * kFmoLsGridMax] block partials of the line-search sums
  FmoState *fmo_state;
  // history
  dao_iter_record *history;  // [k_max]
  DevState *state;
  void *io_scratch;        // small staging buffer for get_vector / hooks ([max(n_vox_pad,n_bl)] 8-byte)
};

struct Ctx {
  // problem
  int32_t n_vox = 0, n_bl = 0, n_beams = 0, n_rows = 0, n_struct = 0;
  int64_t nnz = 0;
  int32_t n_vox_pad = 0;        // n_vox rounded up to a multiple of 128
  int32_t max_rows_per_beam = 0;
  int32_t max_row_len = 0;      // longest leaf row of the context's own MLC tables
  int32_t max_beam_width = 0;   // widest beam in lateral positions (max over rows of row_col0 + row length)
  int32_t n_slices = 0;
  int64_t sell_elems = 0;
  int32_t n_tchunks = 0, n_tsegs = 0;
  dao_options opt{};
  // host copies of small tables
  std::vector<int32_t> beam_row_ptr, row_bl_ptr, row_col0;
  // device
  DevPtrs d{};
  cudaStream_t stream = nullptr;
  int device = 0, n_sm = 0;
  int spmv_grid = 0, master_grid = 0;
  int red_stride = kMaxRedux;   // slots per CTA of the grid reductions (ll_part)
  NewtonLayout nwt{};           // master_method = 2, 3
  size_t master_smem = 0;
  int master_slab = 0, master_stages = 0, master_z_in_smem = 0;
  bool x_in_smem = true;
  bool has_vt = false;          // per-voxel thresholds in use (d.vt)
  int spmv_ring_warps = 0;      // > 0: the TMA-ring SpMV variant with that many warps per CTA
  // host mirror (pinned) of DevState for the once-per-iteration read-back
  DevState *h_state = nullptr;
  // host bookkeeping
  int32_t K = 0;                // pool size as last seen by the host
  bool have_candidate = false;
  bool x_current = false;       // d.x holds the beamlet intensities of the pool's current y (the Newton master writes them)
  bool cand_appended = false;   // the last pricing launch already wrote the candidate into the pool tables
  double objective = 0.0;
  cudaEvent_t ev[8] = {};
  cudaEvent_t ev_state = nullptr;   // marks the copy of the state block (dao_run reads it while later work runs)
  int64_t n_launches = 0;       // kernels launched on the hot path since dao_create (dao_run reports the difference)
  std::vector<double> iter_seconds;   // [apertures added by the last dao_run][6]: per kernel class, when options.timers != 0
  std::string err;
};

// ------------------------------------------------------------------------------------------
// helpers
// ------------------------------------------------------------------------------------------
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

#define DAO_CUDA_OK(ctx, call)                                                            \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
      return DAO_E_CUDA;                                                                  \
    }                                                                                     \
  } while (0)

// Order-independent 64-bit hash of an aperture: beam + sum over its leaf rows of a mixed (row, left, right)
__host__ __device__ __forceinline__ unsigned long long leaf_hash(int32_t m, int32_t l, int32_t r) {
  unsigned long long z = ((unsigned long long)(uint32_t)m << 42) ^ ((unsigned long long)(uint32_t)l << 21) ^ (unsigned long long)(uint32_t)r;
  z += 0x9e3779b97f4a7c15ull;
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}
__host__ __device__ __forceinline__ unsigned long long beam_hash(int32_t b) { return leaf_hash(0x7ffff, b, b); }

// kernels / launchers implemented in the .cu files --------------------------------------------
// dao_setup.cu
struct HostLayout;   // SELL slice table and permutation computed on the host from row_ptr
dao_status setup_build(Ctx *c, const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, void *workspace,
                       size_t workspace_bytes, void *scratch, size_t scratch_bytes);
dao_status setup_sizes(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                       dao_sizes *out, std::string *err);

// dao_spmv.cu
enum SpmvMode { kSpmvObjective = 0, kSpmvPlain = 1, kSpmvColumn = 2, kSpmvPlainUserOrder = 3 };
// `skip` (device, may be null): when *skip != 0 the kernels return at once (device-side loop control).
// kSpmvColumn writes column `a_col` of the dose block A (a_col < 0: column K of the device state, only
// when a candidate is pending), whatever its layout (a_index); `out` is ignored in that mode.
cudaError_t launch_spmv(Ctx *c, SpmvMode mode, const float *x, float *out, const int32_t *skip = nullptr,
                        int32_t a_col = -1);
cudaError_t launch_spmv_t(Ctx *c, const float *g, float *w_out, const int32_t *skip = nullptr);
cudaError_t launch_intensity(Ctx *c);
void spmv_configure(Ctx *c);
// the column SpMV builds the candidate's 0/1 mask itself while it stages x in shared memory (every variant but the
// one that reads x from global memory)
inline bool spmv_builds_mask(const Ctx *c) { return c->spmv_ring_warps > 0 || c->x_in_smem; }

// dao_pricing.cu
cudaError_t launch_pricing(Ctx *c, const float *w, const int32_t *row_bl_ptr, const int32_t *beam_row_ptr,
                           int32_t n_rows, int32_t n_beams, int32_t *left, int32_t *right, double *vstar,
                           double *row_absmax, double *beam_price, double *beam_absmax, int32_t *best_out,
                           bool update_state, int32_t max_row_len = 0 /* 0 = unknown: warp-per-row kernel */);
cudaError_t launch_append_candidate(Ctx *c);
size_t chain_pricing_smem(int32_t max_rows, int32_t width);   // shared memory of k_price_chain
// steps 5-6 without a context, scratch in a fixed array of the library image (dao_price_from_w_static, dao.h)
dao_status price_from_w_static(const float *w, const int32_t *row_bl_ptr, const int32_t *beam_row_ptr, int32_t n_rows,
                               int32_t n_beams, int32_t *left, int32_t *right, double *vstar, double *beam_price,
                               int32_t *best_out, cudaStream_t stream, std::string *err);

// dao_fmo.cu
dao_status fmo_solve(Ctx *c, int32_t max_iter, double tol, bool warm_start, dao_fmo_info *out);

// dao_master.cu (methods 0, 1) -- both dispatch to dao_newton.cu when master_method >= 2
cudaError_t master_configure(Ctx *c);
cudaError_t launch_master(Ctx *c, bool add_candidate);

// dao_newton.cu (methods 2, 3)
NewtonLayout newton_layout(int32_t k_max, int32_t n_vox_pad, int32_t n_struct, bool tc);   // host only, no device query
cudaError_t newton_configure(Ctx *c);
cudaError_t launch_newton(Ctx *c, bool add_candidate);
cudaError_t newton_fill_tile_meta(Ctx *c);   // method 3: writes the meta rows of the tiled dose block (after sid / vt are set)

// Position of (internal voxel i, aperture column k) in the dose block A (floats).  Tiled layouts SPREAD the voxels
// over the tiles: voxel i sits in tile i mod n_tiles at slot i / n_tiles.  The internal voxel order is sorted by the
// length of the voxel's row of D, which clusters the penalised ("active") voxels; spread, every tile -- and with the
// tiles every CTA of the Newton master -- holds the same mix (measured before: the slowest CTA of a pass took 79 us,
// the mean 71 us, and whole tiles of active voxels stalled the conversion pipeline).
__host__ __device__ __forceinline__ size_t a_index(int32_t tile_T, int32_t tile_TP, int64_t tile_stride,
                                                   int32_t n_vox_pad, int32_t n_tiles, int32_t i, int32_t k) {
  if (tile_T == 0) return (size_t)k * (size_t)n_vox_pad + (size_t)i;
  const int32_t slot = i / n_tiles, t = i - slot * n_tiles;
  return (size_t)t * (size_t)tile_stride + (size_t)k * (size_t)tile_TP + (size_t)slot;
}

}  // namespace dao
