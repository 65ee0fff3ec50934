// dao_newton.cu -- step 8 with master_method = 2 and 3: the restricted master problem  min_{y >= 0} F(A y)
// by PROJECTED NEWTON on the free variables.  F is a convex piecewise quadratic
// (eq. 3-5, 9-10), so on a fixed voxel active set its Hessian  H = A^T diag(2 c) A,
// c_j = a_j [z_j < T_j^-] + b_j [z_j > T_j^+],  is exact and a Newton step lands on the minimiser of the
// current piece: 4-5 passes over the dose block A per solve instead of ~120 for gradient projection.
// The paper defers the method of the master to Men et al. 2009 / Bazaraa et al.; the RESULT
// (the optimal value) is unique by convexity, and the stopping test is the one of methods 0/1 and of the
// oracle (reading S2), so parity is unaffected by the choice of method.
//
// ONE persistent cooperative kernel, one CTA per SM, 16 warps (128 registers each).  The dose block is
// stored tiled (NewtonLayout; the voxels are spread over the tiles, a_index): two meta rows (structure ids,
// thresholds) and the K live columns of a tile of T voxels are one contiguous range, fetched by ONE
// cp.async.bulk (1-D TMA) into a stage of a shared-memory ring (issued by lane 0 of an otherwise idle back
// warp).  With all K columns of a tile resident, one pass computes EVERYTHING at a
// trial point y; the warps are specialised:
//  front warps (8):
//   Z  z_j = sum_k y_k A[k][j]                        (fp64, thread per voxel and k-slice)
//   P  F, pi_j = dF/dz_j, s_j = 2 c_j, list of the active voxels (s_j != 0) of the tile
//   W  the fp64 tile  W[k][a] = sqrt(s_a) A[k][a]  (k < K),  W[K][a] = pi_a / sqrt(s_a)  over chunks of AC
//      ACTIVE voxels (fp32 -> fp64 on the integer pipe), double buffered in shared memory
//  back warps (8):
//   H  [H, grad] += W W^T on the fp64 tensor cores (mma.sync m8n8k4 f64: 8x8 blocks, 4 voxels per
//      instruction; every warp owns fixed strips of 1x5 blocks whose accumulators stay in registers for
//      the whole pass).  H[k1][k2] = sum_j A[k1][j] s_j A[k2][j],  grad[k] = sum_j A[k][j] pi_j (row K).
// then one grid reduction of (H, grad, F) through flagged slots (dao_grid_reduce.cuh), and every CTA
// computes the same Newton step on the free set {k : y_k > 0 or grad_k < 0} by an LDL^T factorisation
// in shared memory.  The trial point y + t d (t = 1 unless a bound is hit first) is accepted on
// sufficient decrease of F -- the next pass IS the evaluation -- else t is shortened by the secant
// of phi'(t) = d . grad(y + t d).  All sums fp64 in a fixed order: bit-reproducible.
//
// master_method = 3 is the same kernel template with TC = true: the Hessian on the 5th-generation tensor cores
// (tcgen05.mma kind::tf32 on a hi/lo split of sqrt(s) A, accumulators in TMEM); see the comments at the control
// warps and at pass_tc below, and DESIGN.md sections 6 and 13.
#include "dao_internal.cuh"
#include "dao_ptx.cuh"
#include "dao_grid_reduce.cuh"

#include <math_constants.h>

#include <algorithm>

namespace dao {

constexpr int kNwtStrips = 3;           // strips of H blocks a warp may own: 8 back warps x 3 = the 24 strips of K <= kNewtonMaxK
constexpr int kNwtStripLen = 5;         // 8x8 blocks per strip (one block row, consecutive block columns)
constexpr int kNwtMaxStrips = 48;       // >= sum_I ceil((nb - I) / 4) for nb = 17 (45)
#ifndef DAO_NWT_MIN_STAGES
#define DAO_NWT_MIN_STAGES 2
#endif
constexpr int kNwtMinStages = DAO_NWT_MIN_STAGES;   // ring stages a layout must have (2: bigger W chunks win, measured)
constexpr int kNwtFront = 8;             // front warps: dose, penalty, active list, fp64 tile W
constexpr int kNwtBack = kNW - kNwtFront;   // back warps: H += W W^T on the fp64 tensor cores
constexpr int kNwtFrontThreads = kNwtFront * 32;
// master_method = 3 (tensor cores): tiles of 128 voxels, a GROUP of 4 warps per tile (lane = voxel), 4 groups per CTA.
// A group appends its active voxels to an operand slab of two HALVES of 16 voxels each (filled alternately); a half
// = rows [Wh (64); Wl (64)] x 16 voxels, K-major core matrices (8 rows x 16 bytes): 128 bytes between voxel quads
// (LBO), 512 bytes between groups of 8 rows (SBO).  The tile starts with two META rows (structure ids, per-voxel
// thresholds) so that one bulk copy brings everything a tile needs.
constexpr int kTcT = 128;
constexpr int kTcGroupWarps = kTcT / 32;
constexpr int kTcGroups = kNW / kTcGroupWarps;
constexpr int kTcHV = 16;                // voxels per half = two MMA k-steps
constexpr uint32_t kTcLbo = 128, kTcSbo = (kTcHV / 4) * kTcLbo, kTcHalfBytes = 16 * kTcSbo;
constexpr uint32_t kTcCols = 64 * kTcGroups;   // TMEM columns: one 128 x 64 fp32 accumulator per group
constexpr int kTcMaxK = kNewtonTcMaxK;             // 8 block rows of the augmented Hessian fit the 64 rows of one operand half
constexpr int kTcMaxStages = 12;
constexpr int kNwtMetaRows = 2;
constexpr int kNwtAcc = 7;               // gradient accumulators per thread: rows r, r + 8, ... < 56

struct NewtonParams {
  const float *A;            // tiled dose block
  int32_t n_vox_pad;
  int32_t T, TP;             // tile voxels, column pitch (floats)
  int64_t tile_stride;       // floats between tiles
  int32_t n_tiles;
  int32_t n_stages;
  int32_t stage_bytes;
  int32_t n_red_cap;         // capacity (doubles) of the reduction staging array = slots per CTA
  int32_t lbuf_doubles;      // capacity of the factorisation buffer (also holds the W tile)
  int32_t AC;                // active voxels per chunk of the H phase (power of two)
  int32_t w_doubles;         // doubles per W tile: (8 nb_max + 1) (AC + 4)
  int32_t ks_shift;          // log2 of the k-slices per voxel of the dose loop: T << ks_shift = 256 front threads
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
  // step 1 (eq. 7) of the NEXT column-generation iteration, done here: x_i = sum_{k : i in A_k} y_k
  int32_t n_bl, max_rows;
  const int32_t *bl_row, *row_beam, *beam_row_ptr, *row_bl_ptr, *ap_left, *ap_right;
  float *x;
  int32_t add_candidate;
  int32_t max_iter;
  int32_t k_max;
  double tol;
};

// LDL^T factorisation of the Newton system: threads that take part, column lanes per row
constexpr int kFacThreads = 256, kFacCols = 8;
__device__ __forceinline__ void fac_sync() { asm volatile("bar.sync 7, %0;" ::"n"(kFacThreads) : "memory"); }

// barrier over the front warps
__device__ __forceinline__ void fsync() { asm volatile("bar.sync 2, %0;" ::"n"(kNwtFrontThreads) : "memory"); }
// master_method = 3: every worker warp is a front warp

// fp32 -> fp64 of a finite value >= 0 on the integer pipe (F2F.F64.F32 runs at 16 per clock and SM with ~90
// cycles of latency, measured): exact for normal numbers; +0 maps to 2^-127 -- the dose loop subtracts exactly
// what that adds, the Hessian tile does not care (products with 1e-38 vanish).
__device__ __forceinline__ double cvt_pos(float x) {
  // (b << 29) as a 64-bit product puts b >> 3 into the high word; one IMAD.WIDE with the exponent re-bias added
  const unsigned long long r = (unsigned long long)__float_as_uint(x) * 0x20000000ull + 0x3800000000000000ull;
  return __longlong_as_double((long long)r);
}

// 1 / d for a normal d > 0: hardware seed + two Newton steps (full fp64 accuracy to ~1 ulp, deterministic); the
// IEEE division the compiler emits is a ~30-instruction sequence with a slow path, on the critical path of every pivot
__device__ __forceinline__ double rcp_f64(double d) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  r = fma(r, fma(-d, r, 1.0), r);
  r = fma(r, fma(-d, r, 1.0), r);
  return r;
}

__device__ __forceinline__ double lds_f64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// ---- tcgen05 (5th-generation tensor cores): shared-memory operand descriptors, MMA issue, TMEM access ----
// Operand tiles are K-major ("K" = the contraction index = the voxels of a chunk) without swizzling: a core matrix
// is 8 rows x 16 bytes stored contiguously (row r at +16 r); `lbo` bytes separate core matrices adjacent along the
// voxels, `sbo` bytes separate groups of 8 rows.  One kind::tf32 MMA consumes 8 voxels = two core matrices.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46);   // descriptor version 1 (sm_100), no swizzle
}
// D[tmem] (+)= A[smem] B[smem]^T, M = 128 rows of A, N rows of B (idesc), 8 voxels; fp32 accumulation in TMEM
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrives on `bar` when every MMA issued so far by this thread has completed (implies fence::before_thread_sync)
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// generic-proxy writes to shared memory become visible to the async proxy (the tensor core reads operands through it)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 16 consecutive TMEM columns of this thread's lane (warp w may touch lanes 32 (w % 4) .. + 31 only)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}
__device__ __forceinline__ void sts_f32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }

// rows of the operand tile a worker thread handles are kpar, kpar + kstep, ...: kstep = 512 / AC
__device__ __forceinline__ int kstep_of(int ac_shift) { return kMasterWorkers >> ac_shift; }

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

// 16 warps exactly: a 17th (a dedicated producer warp, as in k_master) would be allocated as 20 warps and cap the
// kernel at 96 registers, which made the compiler serialise the tensor-core loop through one temporary register.
// master_method = 3 (TC = true): every worker warp is a front warp and the Hessian runs on the 5th-generation tensor
// cores -- the front warps write the chunk of active voxels as a TF32 hi/lo operand tile, a 17th CONTROL warp (one
// thread) feeds the A ring and issues tcgen05.mma (accumulators in TMEM for the whole pass); the gradient A^T pi is
// accumulated in fp64 by the threads that write the tile.  Only H (which steers the Newton direction and never enters
// the stopping test) is computed in reduced precision: ~2^-21 relative (3 x TF32), see DESIGN.md section 6.
constexpr int kNwtTcThreads = kMasterWorkers + 96;   // + two control warps and the feeder warp
template <bool TC>
__global__ void __launch_bounds__(TC ? kNwtTcThreads : kMasterWorkers, 1) k_master_newton(NewtonParams p) {
  extern __shared__ __align__(128) unsigned char dyn_smem[];
  __shared__ double y_s[DAO_MAX_APERTURES];        // accepted point
  __shared__ double ytr_s[DAO_MAX_APERTURES];      // trial point of the current pass
  __shared__ double d_s[DAO_MAX_APERTURES];        // Newton direction
  __shared__ double grad_s[DAO_MAX_APERTURES];     // gradient at the accepted point
  __shared__ double dpiv_s[DAO_MAX_APERTURES + 1]; // reciprocals of the pivots of the LDL^T factorisation (an fp64
                                                   // division is ~30 instructions: one per pivot, not one per use)
  __shared__ double xs_s[DAO_MAX_APERTURES + 1];   // solution on the free set
  __shared__ int fr_s[DAO_MAX_APERTURES];          // free variables
  __shared__ unsigned short strip_s[kNwtMaxStrips];  // strip -> (I << 8) | J0, longest strips first
  __shared__ double sc[16];
  __shared__ int si[16];
  __shared__ int wcnt_s[kNW];
  __shared__ volatile int wmeta_s[2];              // per W buffer: columns (multiple of 4) | last chunk of its tile << 16
  __shared__ double fred_s[kNW];
  __shared__ unsigned long long prof_s[kMasterProfSlots];
  __shared__ uint32_t tmem_base_s;                 // TC: base address of the TMEM allocation
  __shared__ volatile int ctrl_cmd_s;              // TC: 1 = another pass follows, 0 = the solve is over
  __shared__ double ycur_s[DAO_MAX_APERTURES];     // TC: the point of the current pass
  __shared__ volatile int smeta_s[kTcGroups][2];   // TC: per half message: bit 0 = it holds voxels, bit 1 = last of the pass
  __shared__ volatile int gcnt_s[kTcGroups][2][kTcGroupWarps];   // TC: active voxels of a tile per warp (double buffered)
  __shared__ volatile int stop_s;                  // TC: the feeder warp stops issuing
  __shared__ volatile int live_s[kTcGroups];       // TC: the group issued an MMA in this pass (its accumulator is live)
  __shared__ volatile int gen_s[16];               // TC: copies issued into ring stage s so far (a group may run several uses of
                                                   // a stage ahead of the feeder: a parity wait alone would alias)
  __shared__ volatile long long total_tiles_s;     // TC: tiles consumed when the solve ended

  constexpr int NF = kNwtFront;                    // front warps (method 2)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int K0 = p.st->K;
  const int cand = p.st->cand_valid;
  const int added = (p.add_candidate && cand) ? 1 : 0;
  const int K = K0 + added;
  if ((p.add_candidate && !added) || K == 0) {     // converged, pool full or empty pool: nothing to solve
    if (blockIdx.x == 0 && tid == 0) { p.st->m_added = 0; p.st->m_iters = 0; p.st->m_passes = 0; }
    // x for the unchanged y (callers rely on the master leaving x current)
    for (int i = (int)blockIdx.x * kMasterWorkers + tid; tid < kMasterWorkers && i < p.n_bl; i += (int)gridDim.x * kMasterWorkers) {
      const int r = p.bl_row[i], b = p.row_beam[r];
      const int m = r - p.beam_row_ptr[b], c = i - p.row_bl_ptr[r];
      double acc = 0.0;
      for (int k = 0; k < K0; ++k) {
        if (p.ap_beam[k] != b) continue;
        if (c >= p.ap_left[k * p.max_rows + m] && c < p.ap_right[k * p.max_rows + m]) acc += p.y[k];
      }
      p.x[i] = (float)acc;
    }
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
  uint64_t *wfull = empty + 8, *wempty = empty + 10;   // the two W buffers (n_stages <= 6)
  // TC: up to 16 stages; per-warp slab barriers; accumulators of a pass complete; next command
  uint64_t *sfull = nullptr, *sempty = nullptr, *acc_full = nullptr, *go = nullptr;
  unsigned char *slabs = nullptr, *cl_s = nullptr;
  double *cpi_s = nullptr, *gpart = nullptr;
  float *csq_s = nullptr, *lh_s = nullptr;
  if constexpr (TC) {
    sfull = reinterpret_cast<uint64_t *>(q); q += 128;
    sempty = reinterpret_cast<uint64_t *>(q); q += 128;
    acc_full = reinterpret_cast<uint64_t *>(q); go = acc_full + 1; q += 128;
    cpi_s = reinterpret_cast<double *>(q); q += kNW * 32 * 8;
    csq_s = reinterpret_cast<float *>(q); q += kNW * 32 * 4;
    cl_s = q; q += kNW * 32;
  }
  StructEntry *stab = reinterpret_cast<StructEntry *>(q); q += align_up_c((size_t)p.n_struct * sizeof(StructEntry), 128);
  if constexpr (TC) { slabs = q; }                 // 16 slabs; idle between the passes: hred, lbuf, lh, gradient partials live here
  double *hred = reinterpret_cast<double *>(q); q += align_up_c((size_t)p.n_red_cap * 8, 128);
  double *lbuf = reinterpret_cast<double *>(q); q += align_up_c((size_t)p.lbuf_doubles * 8, 128);
  if constexpr (TC) {
    lh_s = reinterpret_cast<float *>(q); q += align_up_c((size_t)64 * 65 * 4, 128);
    gpart = reinterpret_cast<double *>(q); q += (size_t)kNW * 64 * 8;
  }
  double *wbuf = lbuf;                             // the two W tiles of the H phase share the factorisation buffer
  const int AC = p.AC, WP = p.AC + 4;              // active voxels per chunk, row pitch of W (4 mod 16: conflict-free)
  const int ac_shift = 31 - __clz(AC);
  const int w_doubles = p.w_doubles;               // doubles per W tile
  double *gs = reinterpret_cast<double *>(q); q += align_up_c((size_t)(T + 4) * 8, 128);
  double *ss = reinterpret_cast<double *>(q); q += align_up_c((size_t)(T + 4) * 8, 128);
  unsigned short *list = reinterpret_cast<unsigned short *>(q);

  if (tid == 0) {
    if constexpr (TC) {
      for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kTcGroupWarps); }
      for (int h = 0; h < 2 * kTcGroups; ++h) { mbar_init(&sfull[h], kTcGroupWarps); mbar_init(&sempty[h], 1); }
      mbar_init(acc_full, 2);
      mbar_init(go, 1);
      stop_s = 0;
      for (int w = 0; w < 16; ++w) gen_s[w] = 0;
    } else {
      for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NF); }
      for (int s = 0; s < 2; ++s) { mbar_init(&wfull[s], NF); mbar_init(&wempty[s], kNwtBack); }
    }
    for (int i = 0; i < kMasterProfSlots; ++i) prof_s[i] = 0ull;
  }
  fence_mbar_init();
  if constexpr (TC) {
    if (warp == kNW) {                             // the control warp owns the TMEM allocation
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_addr(&tmem_base_s)), "r"(kTcCols) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
  }
  __syncthreads();
  if constexpr (TC) tc_fence_after();
  const uint32_t tmem_base = TC ? tmem_base_s : 0u;

  // =============================== control and feeder warps (TC) ================================
  // Warps 16 and 17, one thread each: control warp c serves the groups 2c and 2c + 1.  It takes whichever of their
  // operand halves is ready and issues its two tcgen05.mma (k-steps of 8 voxels) into the accumulator OF THAT GROUP
  // (TMEM columns 64 g ...): the halves of a group arrive in the group's own fixed order and the four accumulators are
  // added in a fixed order afterwards, so the result does not depend on timing.  tcgen05.commit hands the half back
  // to its group; after the last message of both groups the accumulators are published (acc_full).  `go` /
  // ctrl_cmd_s: does another pass follow?
  // Warp 18, one thread: streams the tiles of the CTA's sequence into the ring (one bulk copy per tile: meta rows +
  // the K live columns); it runs ahead into the next pass and is stopped by stop_s.
  if constexpr (TC) {
    if (warp == kNW || warp == kNW + 1) {
      if (lane == 0) {
        const int cw = warp - kNW;
        // instruction descriptor: D = F32, A = B = TF32, both K-major, N = 64, M = 128
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((64u >> 3) << 17) | ((128u >> 4) << 24);
        const uint64_t desc0 = umma_desc(smem_addr(slabs), kTcLbo, kTcSbo);
        const bool cprof = (p.prof != nullptr) && blockIdx.x == 0 && cw == 0;
        uint32_t par = 0u, go_phase = 0u;            // bit (2 gi + b): parity of the next message on half b of group 2 cw + gi
        uint32_t seq = 0u;                           // bit gi: which half the group sends next
        for (;;) {
          uint32_t live = 3u, mma_any = 0u;          // groups that have not sent their last message; groups with an MMA
          long long tcp = cprof ? clock64() : 0ll;
          while (live) {
            bool idle = true;
#pragma unroll
            for (int gi = 0; gi < 2; ++gi) {
              if (!((live >> gi) & 1u)) continue;
              const int g = 2 * cw + gi, b = (seq >> gi) & 1u, hb = 2 * g + b, pb = 2 * gi + b;
              if (!mbar_test_wait(&sfull[hb], (par >> pb) & 1u)) continue;
              idle = false;
              if (cprof) { const long long n_ = clock64(); prof_s[0] += (unsigned long long)(n_ - tcp); tcp = n_; }
              par ^= 1u << pb;
              seq ^= 1u << gi;
              const int meta = smeta_s[g][b];
              if (meta & 1) {
                tc_fence_after();
                const uint64_t d = desc0 + (uint64_t)((uint32_t)hb * (kTcHalfBytes >> 4));
                const uint32_t acc = tmem_base + (uint32_t)g * 64u;
                umma_tf32(acc, d, d, idesc, (mma_any >> gi) & 1u);
                umma_tf32(acc, d + (uint64_t)((2u * kTcLbo) >> 4), d + (uint64_t)((2u * kTcLbo) >> 4), idesc, 1u);
                mma_any |= 1u << gi;
                umma_commit(&sempty[hb]);
              } else {
                mbar_arrive(&sempty[hb]);
              }
              if (meta & 2) live &= ~(1u << gi);
              if (cprof) { const long long n_ = clock64(); prof_s[15] += (unsigned long long)(n_ - tcp); prof_s[7] += 1ull; tcp = n_; }
            }
            if (idle) __nanosleep(32);
          }
          if (mma_any) umma_commit(acc_full);
          else mbar_arrive(acc_full);
          mbar_wait(go, go_phase);
          go_phase ^= 1u;
          if (!ctrl_cmd_s) break;
          tc_fence_after();
        }
      }
      __syncwarp();
      __syncthreads();                               // the final barrier of the workers
      if (warp == kNW)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTcCols) : "memory");
      return;
    }
    if (warp == kNW + 2) {
      if (lane == 0 && ntl > 0) {
        const int Kc = p.st->K + ((p.add_candidate && p.st->cand_valid) ? 1 : 0);
        const uint32_t bytes = (uint32_t)(Kc + kNwtMetaRows) * (uint32_t)TP * 4u;
        RingPos ipc{0, 0u};
        long long c = 0;
        int j = 0;
        bool rv = false, stop = false;
        for (;;) {
          if (c >= NS) {
            while (!mbar_test_wait(&empty[ipc.stage], ipc.phase ^ 1u)) {
              if (stop_s) { stop = true; break; }
              __nanosleep(64);
            }
          }
          if (stop) break;
          const int tile = tb0 + (rv ? ntl - 1 - j : j) * tstep;
          mbar_arrive_expect_tx(&full[ipc.stage], bytes);
          bulk_g2s(ring + (size_t)ipc.stage * p.stage_bytes, p.A + (size_t)tile * (size_t)p.tile_stride, bytes, &full[ipc.stage]);
          __threadfence_block();
          gen_s[ipc.stage] = (int)(c / NS) + 1;
          ipc.advance(NS);
          ++c;
          if (++j == ntl) { j = 0; rv = !rv; }
        }
        // drain: copies issued for tiles that are never consumed must land before the CTA may exit
        for (long long cc = total_tiles_s; cc < c; ++cc) mbar_wait(&full[(int)(cc % NS)], (uint32_t)((cc / NS) & 1));
      }
      __syncwarp();
      __syncthreads();
      return;
    }
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
  Reducer red{p.ll_part, p.ll_result, 0u, p.n_red_cap};
  if (tid == 0) si[7] = (int)*p.epoch;
  wsync();
  red.ep = (uint32_t)si[7];

  // Distribution of the H blocks over the BACK warps.  The upper block triangle is cut into STRIPS of <= 4
  // consecutive blocks of one block row (one A fragment serves the whole strip); the strips, longest first, are
  // dealt to NC classes of back warps in snake order; the NG = 12 / NC warps of a class (groups) share the quads
  // of active voxels.
  if (tid == 0) {
    int n = 0;
    for (int len = kNwtStripLen; len >= 1; --len)
      for (int I = 0; I < nb; ++I)
        for (int J0 = I; J0 < nb; J0 += kNwtStripLen)
          if (min(kNwtStripLen, nb - J0) == len) strip_s[n++] = (unsigned short)((I << 8) | J0);
    si[8] = n;
  }
  wsync();
  const int nstrips = si[8];
  int NC = 1;
  while (NC < kNwtBack && ((nstrips + NC - 1) / NC > kNwtStrips || kNwtBack % NC != 0)) ++NC;
  const int NG = kNwtBack / NC;
  const bool is_front = TC || warp < kNwtFront;
  const int bw = is_front ? 0 : warp - kNwtFront;
  const int cls = bw % NC, grp = bw / NC;
  int nstr = 0;
  int st_offa[kNwtStrips], st_offb[kNwtStrips], st_len[kNwtStrips], st_blk[kNwtStrips];
#pragma unroll
  for (int s = 0; s < kNwtStrips; ++s) {
    const int i = s * NC + ((s & 1) ? NC - 1 - cls : cls);
    st_offa[s] = st_offb[s] = st_len[s] = st_blk[s] = 0;
    if (!is_front && i < nstrips) {
      const int I = strip_s[i] >> 8, J0 = strip_s[i] & 255;
      st_offa[s] = (I * 8 + (lane >> 2)) * WP;
      st_offb[s] = (J0 * 8 + (lane >> 2)) * WP;
      st_len[s] = min(kNwtStripLen, nb - J0);
      st_blk[s] = blk_index(nb, I, J0);
      nstr = s + 1;
    }
  }

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

  RingPos cp{0, 0u};                       // front warps: position in the A stream
  // The A stream is fed by lane 0 of the LAST back warp while it waits for W tiles (issuing a bulk copy costs the
  // issuing thread ~500 cycles: on a front warp that is the critical path of every tile).  Every pass reads the
  // same tiles, odd passes backwards (what was read last is read first: an LRU-like L2 keeps serving the most
  // recent part of A once 4 V K bytes exceed it); the sequence simply continues into the next pass, so the first
  // stages of a pass are in flight while the grid reduces (a pass that never happens is drained before the exit).
  RingPos ip{0, 0u};                       // issue position
  int issued_total = 0, consumed_total = 0, issue_ti = 0;
  bool issue_rev = false;
  const bool is_issuer = tid == kMasterWorkers - 32;
  const uint32_t tile_bytes = (uint32_t)(K + kNwtMetaRows) * (uint32_t)TP * 4u;   // two meta rows + the K live columns
  auto feed = [&]() {                      // issue copies while stages are free; never blocks
    while (ntl > 0) {
      // the stage was used before: all front warps must have released it (try_wait would block for ~0.5 us)
      if (issued_total >= NS && !mbar_test_wait(&empty[ip.stage], ip.phase ^ 1u)) break;
      const int tile = tb0 + (issue_rev ? ntl - 1 - issue_ti : issue_ti) * tstep;
      mbar_arrive_expect_tx(&full[ip.stage], tile_bytes);
      bulk_g2s(ring + (size_t)ip.stage * p.stage_bytes, p.A + (size_t)tile * (size_t)p.tile_stride, tile_bytes,
               &full[ip.stage]);
      ip.advance(NS);
      ++issued_total;
      if (++issue_ti == ntl) { issue_ti = 0; issue_rev = !issue_rev; }
    }
  };
  RingPos wp{0, 0u};                       // position in the two W buffers (front: producing, back: consuming)
  bool w_first_round = true;
  unsigned pass_no = 0;
  const int r8 = lane >> 2, c2 = (lane & 3) * 2;
  const double kTiny = 5.877471754111438e-39;      // 2^-127 = cvt_pos(+0)

  // ---- one pass over A at the point yv: z, F, pi, grad, H -> hred (reduced over the grid) ----
  // Front warps (4): per tile  Z (dose of every voxel, thread = voxel), P (penalty, gradient, curvature weight,
  // list of the active voxels), W (fp64 tile of the active voxels, chunk by chunk into one of two buffers).
  // Back warps (12): per chunk  H += W W^T on the fp64 tensor cores.  The two sides meet only on the mbarriers of
  // the W buffers; the A stage is released by the front warps as soon as the tile's last chunk is converted.
  auto pass = [&](const double *yv) {
    double f_acc = 0.0;
    const bool rev = (pass_no++ & 1u) != 0u;
    if (is_front) {
      // thread = (voxel, k-slice): T * KS = 256 front threads, the KS slices of a voxel in adjacent lanes
      const int ks_shift = p.ks_shift, KS = 1 << ks_shift;
      const int v0 = tid >> ks_shift, zsl = tid & (KS - 1);
      const int nI = (K > zsl) ? (K - zsl + KS - 1) >> ks_shift : 0;      // columns zsl, zsl + KS, ... of this thread
      const int rstep = TP << ks_shift;
      // what the +0 -> 2^-127 of cvt_pos adds to a dose, accumulated exactly like the dose itself
      double zc;
      {
        double c[4] = {0.0, 0.0, 0.0, 0.0};
        int i = 0;
        for (; i + 3 < nI; i += 4) {
#pragma unroll
          for (int u = 0; u < 4; ++u) c[u] = fma(yv[zsl + ((i + u) << ks_shift)], kTiny, c[u]);
        }
#pragma unroll
        for (int u = 0; u < 3; ++u)
          if (i + u < nI) c[u] = fma(yv[zsl + ((i + u) << ks_shift)], kTiny, c[u]);
        zc = (c[0] + c[1]) + (c[2] + c[3]);
      }
      for (int ti = 0; ti < ntl; ++ti) {
        const int tile = tb0 + (rev ? ntl - 1 - ti : ti) * tstep;
        long long tc = prof ? clock64() : 0ll;
#define CYC_MARK(slot)                                    \
  do {                                                    \
    if (prof) {                                           \
      const long long now_ = clock64();                   \
      prof_s[slot] += (unsigned long long)(now_ - tc);    \
      tc = now_;                                          \
    }                                                     \
  } while (0)
        const int vg0 = tile * T + v0;                 // position of the voxel in the tiled order (mz is kept in it)
        const bool in0 = zsl == 0;                       // slots without a voxel carry kNoStruct and zero columns
        mbar_wait(&full[cp.stage], cp.phase);
        CYC_MARK(12);
        // the tile starts with two meta rows: the structure ids and the per-voxel thresholds of its voxels (the front
        // warps used to fetch them from global memory: an exposed L2 round trip per tile)
        const unsigned char *stage = ring + (size_t)cp.stage * p.stage_bytes;
        const float *M = reinterpret_cast<const float *>(stage) + kNwtMetaRows * TP;
        const int sid0 = stage[v0];
        const float vt0 = reinterpret_cast<const float *>(stage)[TP + v0];
        // ---- Z ----
        double z0;
        {
          // four independent chains; the loads of a group of 4 columns are issued together, one group ahead of
          // their use (one or two warps per scheduler cannot hide the shared-memory latency any other way)
          double a[4] = {0.0, 0.0, 0.0, 0.0};
          const float *pa = M + v0 + zsl * TP;
          const double *py = yv + zsl;
          float f[4];
          double yk[4];
          {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const int ii = max(min(u, nI - 1), 0);
              f[u] = pa[(size_t)ii * rstep];
              yk[u] = py[ii << ks_shift];
            }
            int i = 0;
            for (; i + 7 < nI; i += 4) {                 // the next group exists in full: no clamps
              float n[4];
              double yn[4];
              pa += 4 * rstep;
              py += 4 << ks_shift;
#pragma unroll
              for (int u = 0; u < 4; ++u) { n[u] = pa[(size_t)u * rstep]; yn[u] = py[u << ks_shift]; }
#pragma unroll
              for (int u = 0; u < 4; ++u) a[u] = fma(yk[u], cvt_pos(f[u]), a[u]);
#pragma unroll
              for (int u = 0; u < 4; ++u) { f[u] = n[u]; yk[u] = yn[u]; }
            }
            if (i + 3 < nI) {                            // one more full group; its successor is partial
              float n[4];
              double yn[4];
              pa += 4 * rstep;
              py += 4 << ks_shift;
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const int uu = min(u, nI - 1 - (i + 4));     // >= 0 when the partial group is not empty
                n[u] = pa[(size_t)max(uu, 0) * rstep];
                yn[u] = py[max(uu, 0) << ks_shift];
              }
#pragma unroll
              for (int u = 0; u < 4; ++u) a[u] = fma(yk[u], cvt_pos(f[u]), a[u]);
#pragma unroll
              for (int u = 0; u < 4; ++u) { f[u] = n[u]; yk[u] = yn[u]; }
              i += 4;
            }
#pragma unroll
            for (int u = 0; u < 3; ++u)
              if (i + u < nI) a[u] = fma(yk[u], cvt_pos(f[u]), a[u]);
          }
          z0 = ((a[0] + a[1]) + (a[2] + a[3])) - zc;
          // the slices of a voxel sit in adjacent lanes: fixed butterfly
          for (int o = 1; o < KS; o <<= 1) z0 += __shfl_xor_sync(0xffffffffu, z0, o);
        }
        CYC_MARK(13);
        // ---- P ----
        bool act0 = false;
        double sq0 = 0.0, gq0 = 0.0;                             // sqrt(s_j), s_j = 2 c_j; pi_j / sqrt(s_j)
        if (in0) {
          if (sid0 != kNoStruct) {
            StructEntry e = stab[sid0];
            if (p.vt) e.tm = e.tp = (double)vt0;
            const double un = fmax(e.tm - z0, 0.0), ov = fmax(z0 - e.tp, 0.0);
            f_acc += e.a * un * un + e.b * ov * ov;
            const double gv = -2.0 * e.a * un + 2.0 * e.b * ov;
            const double sv = 2.0 * ((un > 0.0 ? e.a : 0.0) + (ov > 0.0 ? e.b : 0.0));
            if (sv != 0.0) {
              act0 = true;
              sq0 = sqrt(sv);
              // pi / s = -(T^- - z) below the band, z - T^+ above it; both sides at once only if T^- > T^+
              gq0 = sq0 * ((un > 0.0 && ov > 0.0) ? gv / sv : (un > 0.0 ? -un : ov));
            }
          }
          p.mz[vg0] = z0;
        }
        const unsigned m0 = __ballot_sync(0xffffffffu, act0);
        if (lane == 0) wcnt_s[warp] = __popc(m0);
        fsync();
        int n_act = 0, off0 = 0;
#pragma unroll
        for (int w = 0; w < kNwtFront; ++w) {
          const int cnt = wcnt_s[w];
          if (w < warp) off0 += cnt;
          n_act += cnt;
        }
        if (act0) {
          const int i = off0 + __popc(m0 & ((1u << lane) - 1u));
          list[i] = (unsigned short)v0; gs[i] = gq0; ss[i] = sq0;
        }
        if (prof) prof_s[11] += (unsigned long long)n_act;
        fsync();
        CYC_MARK(14);
        // ---- W: chunks of AC active voxels.  W[k][a] = sqrt(s_a) A[k][v_a] in fp64, row K: pi_a / sqrt(s_a), so
        //      that W W^T = [H, grad] and both tensor-core operands come straight from W. ----
        int c0 = 0;
        do {
          const int nca = min(AC, n_act - c0), nca4 = (nca + 3) & ~3;
          if (!w_first_round) mbar_spin_wait(&wempty[wp.stage], wp.phase ^ 1u);
          CYC_MARK(5);
          double *wt = wbuf + (size_t)wp.stage * w_doubles;
          if (tid < nca4) wt[(size_t)K * WP + tid] = (tid < nca) ? gs[c0 + tid] : 0.0;
          {
            // thread = (column a, row parity); the voxel of the column is looked up once
            const int a = tid & (AC - 1), kpar = tid >> ac_shift, kstep = kNwtFrontThreads >> ac_shift;
            if (a < nca4) {
              const bool live = a < nca;
              const double sqa = live ? ss[c0 + a] : 0.0;
              const float *src = M + (live ? (int)list[c0 + a] : 0);
              double *dst = wt + a;
              for (int k = kpar; k < K; k += 4 * kstep) {
                float f[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) f[u] = src[(size_t)min(k + u * kstep, K - 1) * TP];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  if (k + u * kstep < K) dst[(size_t)(k + u * kstep) * WP] = sqa * cvt_pos(f[u]);
              }
            }
          }
          c0 += AC;
          if (tid == 0) wmeta_s[wp.stage] = nca4 | (c0 >= n_act ? 0x10000 : 0);
          __syncwarp();
          if (lane == 0) mbar_arrive(&wfull[wp.stage]);
          wp.advance(2);
          if (wp.stage == 0) w_first_round = false;
          CYC_MARK(6);
        } while (c0 < n_act);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[cp.stage]);
        cp.advance(NS);
        ++consumed_total;
      }
#undef CYC_MARK
      wsync();
      PROF_MARK(1);
      for (int gg = 0; gg < NG; ++gg) wsync();         // the back warps add up their blocks
    } else {
      double acc[kNwtStrips][kNwtStripLen][2];
#pragma unroll
      for (int s = 0; s < kNwtStrips; ++s)
#pragma unroll
        for (int m = 0; m < kNwtStripLen; ++m) { acc[s][m][0] = 0.0; acc[s][m][1] = 0.0; }
      for (int ti = 0; ti < ntl; ++ti) {
        bool last;
        do {
          const bool bprof = (p.prof != nullptr) && blockIdx.x == 0 && tid == kNwtFrontThreads;
          long long tb = bprof ? clock64() : 0ll;
          while (!mbar_test_wait(&wfull[wp.stage], wp.phase)) {
            if (is_issuer) feed();
          }
          if (is_issuer) feed();
          if (bprof) { const long long n_ = clock64(); prof_s[0] += (unsigned long long)(n_ - tb); tb = n_; }
          const int meta = wmeta_s[wp.stage];
          last = (meta & 0x10000) != 0;
          const int nq = (meta & 0xffff) >> 2;
          const double *wt = wbuf + (size_t)wp.stage * w_doubles;
          const uint32_t wt_s = smem_addr(wt);
          for (int qd = grp; qd < nq; qd += NG) {
            const uint32_t wq = wt_s + (uint32_t)(qd * 4 + (lane & 3)) * 8u;
#pragma unroll
            for (int s = 0; s < kNwtStrips; ++s) {
              if (s < nstr) {
                // all fragments of the strip are requested before its first tensor-core instruction (left alone,
                // the compiler sinks every load next to its predicated mma and the chain load -> mma runs once
                // per block, 75 cycles instead of 16); a short strip re-reads its last block.  (All strips of a
                // quad at once would need 36 more registers and spills inside this loop.)
                const double fa = lds_f64(wq + (uint32_t)st_offa[s] * 8u);
                double fb[kNwtStripLen];
#pragma unroll
                for (int m = 0; m < kNwtStripLen; ++m)
                  fb[m] = lds_f64(wq + (uint32_t)(st_offb[s] + min(m, st_len[s] - 1) * 8 * WP) * 8u);
                if (st_len[s] == kNwtStripLen) {           // full strip: straight-line tensor-core code
#pragma unroll
                  for (int m = 0; m < kNwtStripLen; ++m) dmma884(acc[s][m][0], acc[s][m][1], fa, fb[m]);
                } else {
#pragma unroll
                  for (int m = 0; m < kNwtStripLen; ++m) {
                    if (m < st_len[s]) dmma884(acc[s][m][0], acc[s][m][1], fa, fb[m]);
                  }
                }
              }
            }
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&wempty[wp.stage]);
          wp.advance(2);
          if (bprof) { prof_s[15] += (unsigned long long)(clock64() - tb); prof_s[7] += 1ull; }
        } while (!last);
      }
      wsync();
      if (is_issuer) feed();                           // every stage is free now: the first tiles of the next pass
      // ---- CTA partial: the groups add their blocks in group order ----
      for (int gg = 0; gg < NG; ++gg) {
        if (grp == gg) {
#pragma unroll
          for (int s = 0; s < kNwtStrips; ++s) {
            if (s < nstr) {
#pragma unroll
              for (int m = 0; m < kNwtStripLen; ++m) {
                if (m < st_len[s]) {
                  double *h = hred + (size_t)(st_blk[s] + m) * 64 + r8 * 8 + c2;
                  if (gg == 0) { h[0] = acc[s][m][0]; h[1] = acc[s][m][1]; }
                  else { h[0] += acc[s][m][0]; h[1] += acc[s][m][1]; }
                }
              }
            }
          }
        }
        wsync();
      }
    }
    {
      const double fs = warp_sum_f64(f_acc);
      if (lane == 0) fred_s[warp] = fs;
    }
    wsync();
    if (tid == 0) {
      double s = 0.0;
      for (int w = 0; w < kNwtFront; ++w) s += fred_s[w];
      hred[nblocks * 64] = s;
    }
    wsync();
    red.ranges(n_red, hred, hred, lbuf);             // the W tiles (= lbuf) are idle between passes
    PROF_MARK(2);
  };

  // ---- the same pass with the Hessian on the 5th-generation tensor cores (master_method = 3) ----
  // No CTA-wide step inside the pass: a tile of 128 voxels belongs to a GROUP of four warps (lane = voxel), the 4
  // groups walk the CTA's tiles independently and meet only on mbarriers.  Per tile and warp:
  //  Z  z_j = sum_k y_k A[k][j]  (fp64, 4 chains);  P  F, pi_j, s_j = 2 c_j, ballot of the active voxels; the four
  //     counts of the group are exchanged through shared memory (one named barrier per tile and group);
  //  W  the group APPENDS its active voxels, in voxel order, to its operand slab: two halves of 16 voxels, rows
  //     [Wh (64); Wl (64)], Wh + Wl = fp32(sqrt(s) A[k][j]) split into two TF32 values (K-major core matrices); lane
  //     (q, r) converts rows r, r + 8, ... of the warp's active voxels q and q + 4 of a chunk of 8 and adds
  //     pi_j A[k][j] to its fp64 gradient accumulators.  A complete half is handed to the control warp (every warp
  //     of the group arrives once per half, after its own writes), which issues [hh; lh] += [Wh; Wl] Wh^T into TMEM.
  // After the last tile the partial half is padded with zeros and sent as the group's last message of the pass; then
  // H = hh + lh + lh^T (the lo x lo term, 2^-22 relative, is dropped), gradient, F -> hred, grid reduction.
  uint32_t acc_phase = 0u;
  long long cbase = 0;                                   // tiles of the earlier passes (position in the A stream)
  unsigned half_base = 0u;                               // halves this group has sent in the earlier passes
  auto pass_tc = [&](const double *yv) {
    double f_acc = 0.0;
    const bool rev = (pass_no++ & 1u) != 0u;
    double gacc[kNwtAcc];
#pragma unroll
    for (int i = 0; i < kNwtAcc; ++i) gacc[i] = 0.0;
    if (tid < K) ycur_s[tid] = yv[tid];
    if (tid < kTcGroups) live_s[tid] = 0;
    wsync();
    const int grp = warp / kTcGroupWarps, wg = warp % kTcGroupWarps;
    unsigned fill = 0u;                                  // active voxels the group has appended in this pass
    {
      // what the +0 -> 2^-127 of cvt_pos adds to a dose, accumulated exactly like the dose itself
      double zc;
      {
        double c[4] = {0.0, 0.0, 0.0, 0.0};
        int k = 0;
        for (; k + 3 < K; k += 4) {
#pragma unroll
          for (int u = 0; u < 4; ++u) c[u] = fma(ycur_s[k + u], kTiny, c[u]);
        }
#pragma unroll
        for (int u = 0; u < 3; ++u)
          if (k + u < K) c[u] = fma(ycur_s[k + u], kTiny, c[u]);
        zc = (c[0] + c[1]) + (c[2] + c[3]);
      }
      const int v = wg * 32 + lane;                      // voxel of the tile
      const int q4 = lane & 3, rp = lane >> 2;           // W: active voxels q4 and q4 + 4 of a chunk, rows rp + 8 i
      const uint32_t slab = smem_addr(slabs) + (uint32_t)grp * 2u * kTcHalfBytes + (uint32_t)rp * 16u;
      unsigned char *my_cl = cl_s + warp * 32;
      double *my_cpi = cpi_s + warp * 32;
      float *my_csq = csq_s + warp * 32;
      // half h (running index of the group) may be written once the message that last used its buffer is consumed
      unsigned verified = half_base;                     // halves below this index are known to be free for writing
      unsigned arrived = half_base;                      // halves below this index: this warp has arrived on sfull
      // this warp is done with every half below `upto` that the group has completed: hand them over
      auto verify_upto = [&](unsigned upto) {
        while (verified < upto) {
          if (verified >= 2u) mbar_wait(&sempty[2 * grp + (verified & 1u)], ((verified >> 1) - 1u) & 1u);
          ++verified;
        }
      };
      auto arrive_upto = [&](unsigned upto) {
        while (arrived < upto) {
          verify_upto(arrived + 1u);                     // the previous phase of this half's barrier must be complete
          fence_async_smem();
          __syncwarp();
          if (lane == 0) {
            if (wg == 0) smeta_s[grp][arrived & 1u] = 1;
            mbar_arrive(&sfull[2 * grp + (arrived & 1u)]);
          }
          ++arrived;
        }
      };
      int tix = 0;
      for (int j = grp; j < ntl; j += kTcGroups, ++tix) {
        const long long c = cbase + j;
        const int stg = (int)(c % NS);
        const uint32_t par = (uint32_t)((c / NS) & 1);
        const int tile = tb0 + (rev ? ntl - 1 - j : j) * tstep;
        long long tc = prof ? clock64() : 0ll;
#define CYC_MARK(slot)                                    \
  do {                                                    \
    if (prof) {                                           \
      const long long now_ = clock64();                   \
      prof_s[slot] += (unsigned long long)(now_ - tc);    \
      tc = now_;                                          \
    }                                                     \
  } while (0)
        while (gen_s[stg] <= (int)(c / NS)) __nanosleep(32);   // the copy of THIS use of the stage has been issued
        mbar_wait(&full[stg], par);
        CYC_MARK(12);
        const unsigned char *stage = ring + (size_t)stg * p.stage_bytes;
        const float *M = reinterpret_cast<const float *>(stage) + kNwtMetaRows * TP;   // column 0 of the tile
        // ---- Z ----
        double z0;
        {
          double a4[4] = {0.0, 0.0, 0.0, 0.0};
          const float *pa = M + v;
          float f[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) f[u] = pa[(size_t)min(u, K - 1) * TP];
          int k = 0;
          for (; k + 7 < K; k += 4) {                    // the next group exists in full
            float n[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) n[u] = pa[(size_t)(k + 4 + u) * TP];
#pragma unroll
            for (int u = 0; u < 4; ++u) a4[u] = fma(ycur_s[k + u], cvt_pos(f[u]), a4[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u) f[u] = n[u];
          }
          if (k + 3 < K) {                               // one more full group; its successor is partial
            float n[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) n[u] = pa[(size_t)min(k + 4 + u, K - 1) * TP];
#pragma unroll
            for (int u = 0; u < 4; ++u) a4[u] = fma(ycur_s[k + u], cvt_pos(f[u]), a4[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u) f[u] = n[u];
            k += 4;
          }
#pragma unroll
          for (int u = 0; u < 3; ++u)
            if (k + u < K) a4[u] = fma(ycur_s[k + u], cvt_pos(f[u]), a4[u]);
          z0 = ((a4[0] + a4[1]) + (a4[2] + a4[3])) - zc;
        }
        CYC_MARK(13);
        // ---- P ----
        bool act0 = false;
        float sq0 = 0.f;
        double gv0 = 0.0;                                 // sqrt(s_j) (fp32), pi_j
        {
          const int sid0 = stage[v];
          if (sid0 != kNoStruct) {
            StructEntry e = stab[sid0];
            if (p.vt) e.tm = e.tp = (double)reinterpret_cast<const float *>(stage)[TP + v];
            const double un = fmax(e.tm - z0, 0.0), ov = fmax(z0 - e.tp, 0.0);
            f_acc += e.a * un * un + e.b * ov * ov;
            const double sv = 2.0 * ((un > 0.0 ? e.a : 0.0) + (ov > 0.0 ? e.b : 0.0));
            if (sv != 0.0) {
              act0 = true;
              gv0 = -2.0 * e.a * un + 2.0 * e.b * ov;
              sq0 = sqrtf((float)sv);
            }
          }
          p.mz[(size_t)tile * T + v] = z0;
        }
        const unsigned m0 = __ballot_sync(0xffffffffu, act0);
        const int n_w = __popc(m0);
        if (act0) {
          const int i = __popc(m0 & ((1u << lane) - 1u));
          my_cl[i] = (unsigned char)v; my_cpi[i] = gv0; my_csq[i] = sq0;
        }
        if (lane == 0) gcnt_s[grp][tix & 1][wg] = n_w;
        asm volatile("bar.sync %0, %1;" ::"r"(3 + grp), "n"(kTcGroupWarps * 32) : "memory");
        unsigned off_w = 0u, n_t = 0u;
#pragma unroll
        for (int w = 0; w < kTcGroupWarps; ++w) {
          const unsigned cn = (unsigned)gcnt_s[grp][tix & 1][w];
          if (w < wg) off_w += cn;
          n_t += cn;
        }
        if (prof) prof_s[11] += (unsigned long long)n_t;
        CYC_MARK(14);
        // ---- W: this warp's active voxels go to the positions fill + off_w ... of the group's stream ----
        const unsigned pos_w = fill + off_w;
        const unsigned done_after = half_base + (fill + n_t) / kTcHV;     // halves complete once this tile is in
        for (int c0 = 0; c0 < n_w; c0 += 8) {
          const unsigned h_first = half_base + (pos_w + c0) / kTcHV;
          const unsigned h_last = half_base + (pos_w + min(c0 + 7, n_w - 1)) / kTcHV;
          arrive_upto(min(h_first, done_after));
          verify_upto(h_last + 1u);
          CYC_MARK(5);
          const int a0 = c0 + q4, a1 = a0 + 4;
          const bool l0 = a0 < n_w, l1 = a1 < n_w;
          const float s0 = l0 ? my_csq[a0] : 0.f, s1 = l1 ? my_csq[a1] : 0.f;
          const double p0 = l0 ? my_cpi[a0] : 0.0, p1 = l1 ? my_cpi[a1] : 0.0;
          const float *src0 = M + (l0 ? (int)my_cl[a0] : 0), *src1 = M + (l1 ? (int)my_cl[a1] : 0);
          const unsigned ps0 = pos_w + a0, ps1 = pos_w + a1;             // position in the group's stream
          const uint32_t o0 = slab + (((half_base + ps0 / kTcHV) & 1u) ? kTcHalfBytes : 0u) + ((ps0 % kTcHV) >> 2) * kTcLbo + (ps0 & 3u) * 4u;
          const uint32_t o1 = slab + (((half_base + ps1 / kTcHV) & 1u) ? kTcHalfBytes : 0u) + ((ps1 % kTcHV) >> 2) * kTcLbo + (ps1 & 3u) * 4u;
          float f0[kNwtAcc], f1[kNwtAcc];
#pragma unroll
          for (int i = 0; i < kNwtAcc; ++i) {
            const size_t ro = (size_t)min(rp + 8 * i, K - 1) * TP;
            f0[i] = src0[ro];
            f1[i] = src1[ro];
          }
#pragma unroll
          for (int i = 0; i < kNwtAcc; ++i) {
            if (rp + 8 * i < K) {
              const float w0 = s0 * f0[i], w1 = s1 * f1[i];
              const float h0 = tf32_rna(w0), h1 = tf32_rna(w1);
              if (l0) {
                sts_f32(o0 + (uint32_t)i * kTcSbo, h0);
                sts_f32(o0 + (uint32_t)(i + 8) * kTcSbo, tf32_rna(w0 - h0));
              }
              if (l1) {
                sts_f32(o1 + (uint32_t)i * kTcSbo, h1);
                sts_f32(o1 + (uint32_t)(i + 8) * kTcSbo, tf32_rna(w1 - h1));
              }
              gacc[i] = fma(p0, cvt_pos(f0[i]), gacc[i]);
              gacc[i] = fma(p1, cvt_pos(f1[i]), gacc[i]);
            }
          }
          CYC_MARK(6);
        }
        fill += n_t;
        arrive_upto(done_after);                         // every half this tile completed (also those without a voxel of this warp)
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[stg]);
      }
      // ---- last message of the pass: the partial half, its unused voxels zeroed (warp 0 of the group) ----
      {
        const unsigned h = half_base + fill / kTcHV, used = fill % kTcHV;
        verify_upto(h + 1u);
        if (wg == 0 && used > 0u) {
          for (unsigned cc = used + (unsigned)q4; cc < (unsigned)kTcHV; cc += 4u) {
            const uint32_t o = slab + ((h & 1u) ? kTcHalfBytes : 0u) + (cc >> 2) * kTcLbo + (cc & 3u) * 4u;
#pragma unroll
            for (int i = 0; i < kNwtAcc; ++i) {
              if (rp + 8 * i < K) {
                sts_f32(o + (uint32_t)i * kTcSbo, 0.f);
                sts_f32(o + (uint32_t)(i + 8) * kTcSbo, 0.f);
              }
            }
          }
        }
        fence_async_smem();
        __syncwarp();
        if (lane == 0) {
          if (wg == 0) smeta_s[grp][h & 1u] = (used > 0u ? 1 : 0) | 2;
          mbar_arrive(&sfull[2 * grp + (h & 1u)]);
        }
        half_base = h + 1u;
        if (fill > 0u && wg == 0 && lane == 0) live_s[grp] = 1;   // the group's accumulator is live in this pass
      }
#undef CYC_MARK
    }
    cbase += ntl;
    // the slab area is recycled below (lh, gradient partials, hred): every warp must be past its last write
    wsync();
    PROF_MARK(1);
    mbar_wait(acc_full, acc_phase);
    acc_phase ^= 1u;
    tc_fence_after();
    // ---- gradient: lanes (q, r) -> r; rows r + 8 i.  Per-warp partials, added in warp order below ----
#pragma unroll
    for (int i = 0; i < kNwtAcc; ++i) {
      double g = gacc[i];
      g += __shfl_xor_sync(0xffffffffu, g, 1);
      g += __shfl_xor_sync(0xffffffffu, g, 2);
      if ((lane & 3) == 0) gpart[warp * 64 + (lane >> 2) + 8 * i] = g;
    }
    {
      const double fs = warp_sum_f64(f_acc);
      if (lane == 0) fred_s[warp] = fs;
    }
    // ---- accumulators: TMEM lanes 0..63 hold hh, lanes 64..127 lh (columns 0..63); lh goes through shared memory ----
    const int lq = warp & 3, cs0 = (warp >> 2) * 16;   // lane quarter, first of the 16 columns of this warp
    const int row = 32 * (lq & 1) + lane;
    bool any_h = false;
#pragma unroll
    for (int g = 0; g < kTcGroups; ++g) any_h = any_h || (live_s[g] != 0);
    if (any_h && lq >= 2) {
      float acc[16];
#pragma unroll
      for (int jj = 0; jj < 16; ++jj) acc[jj] = 0.f;
#pragma unroll
      for (int g = 0; g < kTcGroups; ++g) {
        if (live_s[g]) {
          float vv[16];
          tmem_ld16(tmem_base + ((uint32_t)(32 * lq) << 16) + (uint32_t)(64 * g + cs0), vv);
#pragma unroll
          for (int jj = 0; jj < 16; ++jj) acc[jj] += vv[jj];
        }
      }
#pragma unroll
      for (int jj = 0; jj < 16; ++jj) lh_s[row * 65 + cs0 + jj] = acc[jj];
    }
    wsync();
    if (lq < 2 && row - lane < 8 * nb) {               // warp-uniform: tcgen05.ld is a warp-wide instruction
      double hh[16];
#pragma unroll
      for (int jj = 0; jj < 16; ++jj) hh[jj] = 0.0;
#pragma unroll
      for (int g = 0; g < kTcGroups; ++g) {
        if (live_s[g]) {
          float vv[16];
          tmem_ld16(tmem_base + ((uint32_t)(32 * lq) << 16) + (uint32_t)(64 * g + cs0), vv);
#pragma unroll
          for (int jj = 0; jj < 16; ++jj) hh[jj] += (double)vv[jj];
        }
      }
#pragma unroll
      for (int jj = 0; jj < 16; ++jj) {
        const int col = cs0 + jj;
        if (row < 8 * nb && col < 8 * nb && (row >> 3) <= (col >> 3)) {
          double h = 0.0;
          if (row < K && col < K) {
            if (any_h) h = (hh[jj] + (double)lh_s[row * 65 + col]) + (double)lh_s[col * 65 + row];
          } else if (col == K && row < K) {            // gradient column of the augmented matrix
            double g = 0.0;
            for (int w = 0; w < kNW; ++w) g += gpart[w * 64 + row];
            h = g;
          }
          hred[(size_t)blk_index(nb, row >> 3, col >> 3) * 64 + (row & 7) * 8 + (col & 7)] = h;
        }
      }
    }
    tc_fence_before();
    if (tid == 0) {
      double s = 0.0;
      for (int w = 0; w < kNW; ++w) s += fred_s[w];
      hred[nblocks * 64] = s;
    }
    wsync();
    red.ranges(n_red, hred, hred, lbuf);
    PROF_MARK(2);
  };

  // ---- the first pass evaluates everything at the warm start (previous optimum, new column at 0), every later
  //      one at a trial point.  pass() has ONE call site: inlined several times the kernel outgrew the instruction
  //      cache and everything that runs once per iteration ran from L2 (5x slower, measured). ----
  int passes = 0, iters = 0, hit_max = 0, nbt = 0, stall = 0;
  bool have_dir = false, restoring = false;
  double F = 0.0, t_step = 0.0, slope0 = 0.0, kkt = 0.0, pgmax = 0.0;
  const double *cur = y_s;

  for (;;) {
    if constexpr (TC) {
      if (passes > 0 && tid == 0) { ctrl_cmd_s = 1; mbar_arrive(go); }   // the control warp starts the next pass
      pass_tc(cur);
    } else {
      pass(cur);
    }
    ++passes;
    if (passes == 1) F = hred[nblocks * 64];
    if (restoring) have_dir = false;
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
      cur = ytr_s;
      continue;
    }
    if (verdict == 2) {                                    // no acceptable step: restore z = A y and stop
      hit_max = 1;
      restoring = true;
      cur = y_s;
      continue;
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
      PROF_MARK(8);
      if (prof) ++prof_s[10];
      // Right-looking LDL^T, one column per step, by the first kFacThreads threads.  Column j keeps the unscaled
      // c_ij = l_ij d_j.  Look-ahead: the thread that updates the NEXT pivot (j + 1, j + 1) does so first and stores
      // its reciprocal, so that a step starts with one shared-memory load.  Every element receives its updates in the
      // order j = 0, 1, ...  Measured at K = 50 (B200): 19.7 us with 256 threads, 24 us with 128, 61 us with 32 -- the
      // same as the blocked variant it replaces (8 columns per step, 3 CTA-wide barriers: 19.5 us), faster at small K
      // (3.6 vs 4.7 us at K = 11).  What bounds it is the chain pivot -> reciprocal -> next pivot: ~8 dependent fp64
      // operations per column.
      if (tid < kFacThreads) {
        const int r = tid / kFacCols, cl = tid % kFacCols;
        if (tid == 0) {
          double d0 = lbuf[lidx(0, 0)];
          if (!(d0 > ridge)) d0 = ridge;
          dpiv_s[0] = rcp_f64(d0);
        }
        fac_sync();
        for (int j = 0; j < nf; ++j) {
          const double inv = dpiv_s[j];
          if (tid == 0 && j + 1 < nf) {                        // look-ahead: pivot j + 1
            const double c = lbuf[lidx(j + 1, j)];
            double d1 = fma(-c * inv, c, lbuf[lidx(j + 1, j + 1)]);
            lbuf[lidx(j + 1, j + 1)] = d1;
            if (!(d1 > ridge)) d1 = ridge;
            dpiv_s[j + 1] = rcp_f64(d1);
          }
          for (int i = j + 1 + r; i <= nf; i += kFacThreads / kFacCols) {
            const double f = -lbuf[lidx(i, j)] * inv;
            const int kend = (i == j + 1) ? j : min(i, nf - 1);    // element (j + 1, j + 1) is done by the look-ahead
            double *rowi = lbuf + lidx(i, 0);
            // batches of 4 columns: all loads, then the arithmetic, then the stores (element by element the
            // compiler must keep a store ahead of the next loads: ~50 cycles per element instead of ~15)
            for (int k0 = j + 1 + cl; k0 <= kend; k0 += 4 * kFacCols) {
              double a[4], c[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const int k = min(k0 + u * kFacCols, kend);
                a[u] = rowi[k];
                c[u] = lbuf[lidx(k, j)];
              }
#pragma unroll
              for (int u = 0; u < 4; ++u)
                if (k0 + u * kFacCols <= kend) rowi[k0 + u * kFacCols] = fma(f, c[u], a[u]);
            }
          }
          fac_sync();
        }
      }
      wsync();
      PROF_MARK(9);
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
          const double xk = uk * dpiv_s[k];
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
    cur = ytr_s;
  }
  wsync();

  // ---- publish ----
  // drain: every issued stage must have landed before the CTA may exit
  if constexpr (TC) {
    if (tid == 0) {                                          // the feeder drains the ring, a control warp frees the TMEM
      total_tiles_s = cbase;
      __threadfence_block();
      stop_s = 1;
      ctrl_cmd_s = 0;
      mbar_arrive(go);
    }
  } else {
    if (is_issuer) si[9] = issued_total;
    wsync();
    if (tid == 0) {
      for (const int n_issued = si[9]; consumed_total < n_issued; ++consumed_total) {
        mbar_wait(&full[cp.stage], cp.phase);
        cp.advance(NS);
      }
    }
  }
  // beamlet intensities of the new plan (every CTA a slice; same arithmetic as k_intensity: fp64 sum in pool order)
  for (int i = (int)blockIdx.x * kMasterWorkers + tid; i < p.n_bl; i += (int)gridDim.x * kMasterWorkers) {
    const int r = p.bl_row[i], b = p.row_beam[r];
    const int m = r - p.beam_row_ptr[b], c = i - p.row_bl_ptr[r];
    double acc = 0.0;
    for (int k = 0; k < K; ++k) {
      if (p.ap_beam[k] != b) continue;
      if (c >= p.ap_left[k * p.max_rows + m] && c < p.ap_right[k * p.max_rows + m]) acc += y_s[k];
    }
    p.x[i] = (float)acc;
  }
  if (blockIdx.x == 0) {
    if (tid < K) p.y[tid] = y_s[tid];
    if (tid == 0) {
      *p.epoch = red.ep;
      if (p.prof) {
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
  __syncthreads();       // nobody leaves before the ring is drained
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
static size_t newton_fixed_smem(int32_t k_max, int32_t T, int32_t n_struct, int32_t n_red, int32_t lbuf_doubles) {
  return 128 + 128 + align_up((size_t)std::max(n_struct, 1) * sizeof(StructEntry), 128) + align_up((size_t)n_red * 8, 128) +
         align_up((size_t)lbuf_doubles * 8, 128) + 2 * align_up((size_t)(T + 4) * 8, 128) +
         align_up((size_t)(T + 8) * 2, 128);
}

NewtonLayout newton_layout(int32_t k_max, int32_t n_vox_pad, int32_t n_struct, bool tc) {
  NewtonLayout L;
  L.nb_max = (k_max + 1 + 7) / 8;
  L.n_red = L.nb_max * (L.nb_max + 1) / 2 * 64 + 8;
  // 227 KB opt-in maximum per CTA on sm_100; ~9 KB of static tables, 1 KB reserved by the system
  const size_t budget = (size_t)227 * 1024 - (size_t)11 * 1024;
  if (tc && k_max <= kTcMaxK) {
    // master_method = 3: tiles of 128 voxels (a group of four warps each); a stage = the two meta rows (structure
    // ids, per-voxel thresholds) + the k_max columns of a tile; as many stages as fit beside the operand slabs (whose
    // 64 KB also hold hred, the factorisation buffer, lh and the gradient partials between the passes)
    L.tc = 1;
    L.kp = 64; L.lbo = (int32_t)kTcLbo; L.sbo = (int32_t)kTcSbo; L.w_bytes = (int32_t)kTcHalfBytes; L.tmem_cols = (int32_t)kTcCols;
    L.meta_rows = kNwtMetaRows;
    L.T = kTcT; L.TP = kTcT + 4; L.AC = 64;
    L.lbuf_doubles = std::max((k_max + 1) * (k_max + 2) / 2 + 8, kNW * 32);
    L.stage_bytes = (int32_t)align_up((size_t)(k_max + kNwtMetaRows) * L.TP * 4, 128);
    const size_t recycled = align_up((size_t)L.n_red * 8, 128) + align_up((size_t)L.lbuf_doubles * 8, 128) +
                            align_up((size_t)64 * 65 * 4, 128) + (size_t)kNW * 64 * 8;
    const size_t fixed = 5 * 128 + (size_t)kNW * 32 * 13 + align_up((size_t)std::max(n_struct, 1) * sizeof(StructEntry), 128) +
                         std::max(recycled, (size_t)kTcGroups * 2 * kTcHalfBytes);
    int32_t stages = 2;
    while (stages < kTcMaxStages && fixed + (size_t)(stages + 1) * L.stage_bytes <= budget) ++stages;
    L.n_stages = stages;
    L.smem = fixed + (size_t)stages * L.stage_bytes;
    L.n_tiles = (n_vox_pad + L.T - 1) / L.T;
    L.tile_stride = (int64_t)(k_max + kNwtMetaRows) * L.TP;
    return L;
  }
  static const int32_t cand_t[] = {256, 128, 64, 32};        // T x k-slices = 256 front threads
  static const int32_t cand_ac[] = {64, 32, 16};
  for (int32_t T : cand_t) {
    for (int32_t AC : cand_ac) {
      const int32_t lbuf = std::max((k_max + 1) * (k_max + 2) / 2 + 8, 2 * (8 * L.nb_max + 1) * (AC + 4));
      const int32_t TP = T + 4;
      const int32_t stage = (int32_t)align_up((size_t)(k_max + kNwtMetaRows) * TP * 4, 128);
      const size_t fixed = newton_fixed_smem(k_max, T, n_struct, L.n_red, lbuf);
      if (fixed + (size_t)kNwtMinStages * stage > budget && !(AC == 16 && T == 32)) continue;
      if (AC == 16 && T > 32) continue;                      // rather a smaller tile than 4-quad chunks
      int32_t stages = 2;
      while (stages < 6 && fixed + (size_t)(stages + 1) * stage <= budget) ++stages;
      L.T = T; L.TP = TP; L.stage_bytes = stage; L.n_stages = stages;
      L.AC = AC; L.lbuf_doubles = lbuf;
      L.smem = fixed + (size_t)stages * stage;
      break;
    }
    if (L.T) break;
  }
  L.meta_rows = kNwtMetaRows;
  L.n_tiles = (n_vox_pad + L.T - 1) / L.T;
  L.tile_stride = (int64_t)(k_max + kNwtMetaRows) * L.TP;
  return L;
}

// master_method = 3: the structure id and the threshold of every voxel of a tile, in the tile's two meta rows
__global__ void k_newton_tile_meta(float *A, int32_t n_tiles, int32_t T, int32_t TP, int64_t tile_stride, const uint8_t *sid,
                                   const float *vt, int32_t n_vox_pad) {
  const int pos = (int)(blockIdx.x * blockDim.x + threadIdx.x);
  if (pos >= n_tiles * T) return;
  const int t = pos / T, v = pos - t * T;
  const int i = v * n_tiles + t;                     // the voxel at slot v of tile t (a_index)
  float *tile = A + (size_t)t * (size_t)tile_stride;
  reinterpret_cast<uint8_t *>(tile)[v] = (i < n_vox_pad) ? sid[i] : (uint8_t)kNoStruct;
  tile[TP + v] = (vt != nullptr && i < n_vox_pad) ? vt[i] : 0.f;
}

cudaError_t newton_fill_tile_meta(Ctx *c) {
  const NewtonLayout &L = c->nwt;
  if (!L.meta_rows) return cudaSuccess;
  const int n = L.n_tiles * L.T;
  k_newton_tile_meta<<<(n + 255) / 256, 256, 0, c->stream>>>(c->d.A, L.n_tiles, L.T, L.TP, L.tile_stride, c->d.sid,
                                                           c->has_vt ? c->d.vt : nullptr, c->n_vox_pad);
  return cudaGetLastError();
}

cudaError_t newton_configure(Ctx *c) {
  c->master_grid = std::min(c->n_sm, kMasterMaxGrid);
  if (c->opt.reserved & 16) c->master_grid = std::min(c->master_grid, 8);   // test hook: many tiles per CTA on small inputs
  const NewtonLayout &L = c->nwt;
  const void *fn = L.tc ? (const void *)k_master_newton<true> : (const void *)k_master_newton<false>;
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);
  if (e != cudaSuccess) return e;
  int nbk = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nbk, fn, L.tc ? kNwtTcThreads : kMasterWorkers, L.smem);
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
  p.lbuf_doubles = L.lbuf_doubles;
  p.AC = L.AC;
  p.w_doubles = (8 * L.nb_max + 1) * (L.AC + 4);
  p.ks_shift = 0;
  while ((L.T << p.ks_shift) < (L.tc ? kMasterWorkers : kNwtFrontThreads)) ++p.ks_shift;

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
  p.n_bl = c->n_bl; p.max_rows = c->max_rows_per_beam;
  p.bl_row = c->d.bl_row; p.row_beam = c->d.row_beam; p.beam_row_ptr = c->d.beam_row_ptr; p.row_bl_ptr = c->d.row_bl_ptr;
  p.ap_left = c->d.ap_left; p.ap_right = c->d.ap_right; p.x = c->d.x;
  c->x_current = true;                     // the kernel leaves x consistent with the y it returns
  p.add_candidate = add_candidate ? 1 : 0;
  p.max_iter = c->opt.master_max_iter;
  p.k_max = c->opt.k_max;
  p.tol = c->opt.master_tol;
  void *args[] = {&p};
  ++c->n_launches;
  if (L.tc)
    return cudaLaunchCooperativeKernel((void *)k_master_newton<true>, dim3(c->master_grid), dim3(kNwtTcThreads), args,
                                       L.smem, c->stream);
  return cudaLaunchCooperativeKernel((void *)k_master_newton<false>, dim3(c->master_grid), dim3(kMasterWorkers), args,
                                     L.smem, c->stream);
}

}  // namespace dao
