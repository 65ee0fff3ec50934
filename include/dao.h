/*
 * dao.h -- C ABI of the B200-native hot path of column-generation direct aperture optimisation
 * (DAO) after Men, Jia & Jiang, arXiv 1003.5402.  Citations are PAPER.md:<line> (+ equation).
 *
 * The library computes, entirely in hand-written CUDA kernels for sm_100a:
 *   1. beamlet intensities   x_i = sum_{k : i in A_k} y_k                  PAPER.md:96-98 (eq. 7)
 *   2. voxel dose            z_j = sum_i D_ij x_i                           PAPER.md:65    (eq. 1, 2)
 *   3. objective + gradient  F(z), pi_j = dF/dz_j                           PAPER.md:75-83 (eq. 3-5),
 *                                                                           :246-254 (eq. 9-10), :136
 *   4. beamlet gradient      w_i = sum_j D_ij pi_j                          PAPER.md:138-140 (eq. 8)
 *   5. row pricing           per MLC leaf row the contiguous interval with the most negative sum
 *                            of w (ties: smallest left leaf, then smallest right leaf)
 *                                                                           PAPER.md:140-167
 *   6. beam selection        price_b = sum of the row minima of beam b; b* = argmin_b (ties: smallest b)
 *                                                                           PAPER.md:169
 *   7. aperture dose column  a_K = sum_{i in A_K} D_i.                      PAPER.md:69 (eq. 2)
 *   8. restricted master     min_{y >= 0} F(A y): gradient projection as the paper names it (methods 0, 1) or
 *                            projected Newton to the same unique optimum (methods 2, 3; 2 is the default)
 *                                                                           PAPER.md:114, 134
 *   9. the column-generation loop over 1-8
 *
 * Conventions
 *   - D is passed voxel-major: row j = voxel, column i = beamlet (the paper writes D_ij with i the
 *     beamlet).  Values fp32, indices int32.
 *   - Beamlets are numbered beam-major, then MLC leaf row, then left to right, so each leaf row
 *     is a contiguous range of beamlet ids [row_bl_ptr[r], row_bl_ptr[r+1]).
 *   - Leaf positions are 0-based half-open [left, right) column offsets inside the leaf row: the
 *     open beamlets of row r are row_bl_ptr[r]+left .. row_bl_ptr[r]+right-1.  In the paper's
 *     1-based notation left = l*, right = r* - 1 (open beamlets l*+1 .. r*-1, PAPER.md:140,
 *     156-165).  A closed row is (0, 0) (the paper's initial (l*, r*) = (0, 1)).
 *   - Every function returns a dao_status; nothing throws, aborts or prints.  Functions that
 *     return host scalars synchronise the context's stream once, at their end; dao_run
 *     synchronises once per column-generation iteration.
 *   - The library never allocates device memory: the caller (PyTorch in the Python binding)
 *     provides one persistent workspace and one create-time scratch buffer whose sizes
 *     dao_workspace_bytes reports, and the CUDA stream all work is issued on.
 *   - Inputs are only read during dao_workspace_bytes / dao_create; nothing of the caller's is
 *     referenced afterwards.  Pointers flagged DAO_MEM_DEVICE must be device pointers valid on
 *     the current device; DAO_MEM_HOST pointers are ordinary host memory (pinned or pageable).
 *   - A context is not thread-safe and is bound to the stream given at creation.
 *   - There is no CPU fallback: without a CUDA device every call that needs one fails with
 *     DAO_E_CUDA.
 */
#ifndef DAO_H_
#define DAO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dao_ctx dao_ctx;   /* opaque; one per plan */

typedef enum {
  DAO_OK = 0,
  DAO_E_ARG = 1,          /* null pointer, negative size, non-finite / negative value, bad option */
  DAO_E_SHAPE = 2,        /* inconsistent sizes, non-monotone pointers, index out of range, capacity too small */
  DAO_E_CUDA = 3,         /* a CUDA call failed; text in dao_last_error */
  DAO_E_ALLOC = 4,        /* workspace / scratch too small or misaligned */
  DAO_E_STATE = 5,        /* call not valid in the context's current state */
  DAO_E_UNSUPPORTED = 6   /* nnz >= 2^31, more than 255 structures, more than DAO_MAX_APERTURES apertures */
} dao_status;

typedef enum { DAO_MEM_HOST = 0, DAO_MEM_DEVICE = 1 } dao_memspace;

#define DAO_MAX_APERTURES 128      /* upper bound on dao_options.k_max */

/* The beamlet dose-deposition matrix D_ij, CSR, rows = voxels, columns = beamlets. */
typedef struct {
  int32_t n_vox, n_bl;
  int64_t nnz;               /* < 2^31 */
  const int32_t *row_ptr;    /* [n_vox+1], row_ptr[0] = 0, non-decreasing, row_ptr[n_vox] = nnz */
  const int32_t *col_idx;    /* [nnz], strictly ascending inside a row, in [0, n_bl) */
  const float *val;          /* [nnz], finite, >= 0 */
  dao_memspace mem;          /* where the three arrays live */
} dao_csr;

/* MLC geometry: which beamlets form a leaf row, which leaf rows form a beam. */
typedef struct {
  int32_t n_beams, n_rows;
  const int32_t *beam_row_ptr;   /* [n_beams+1] host, into leaf rows; beam_row_ptr[n_beams] = n_rows */
  const int32_t *row_bl_ptr;     /* [n_rows+1]  host, into beamlets;  row_bl_ptr[n_rows] = n_bl */
  const int32_t *row_col0;       /* optional [n_rows] host (NULL = all 0): lateral position, in beamlet widths, of
                                    the first beamlet of every leaf row (rows are contiguous hulls that need not
                                    start at the same place; consecutive rows of a beam are physically adjacent).
                                    >= 0.  Only read by MLC modes that couple rows (DAO_MLC_JAWS_ONLY) */
} dao_mlc;

/* MLC deliverability rule of the pricing sub-problem ("standard consecutiveness, interdigitation,
 * connectedness and jaws-only delivery"; the paper shows results, and prints an algorithm, for the first only). */
typedef enum {
  DAO_MLC_CONSECUTIVE = 0,   /* every leaf row opens one contiguous interval, rows independent */
  DAO_MLC_INTERDIGITATION = 2,  /* reading J2: leaf states (a, b) = lateral tip positions of the left and right leaf
                                of a row (open cells [a, b), closed when a == b, an open row stays inside its own
                                beamlets, a closed pair parks anywhere); for physically adjacent rows m, m+1 no leaf
                                passes the opposing leaf of the neighbour: a_m <= b_{m+1} and a_{m+1} <= b_m */
  DAO_MLC_CONNECTED = 3,     /* reading J3: the open rows are consecutive and the open intervals of adjacent open
                                rows share at least one lateral position; closed rows are free.  Modes 2 and 3 are
                                solved by a dynamic programme over the rows; only the optimal VALUE is unique */
  DAO_MLC_JAWS_ONLY = 1      /* reading J1 of DESIGN.md: the aperture is a rectangle -- consecutive leaf rows m1..m2
                                of the beam all opened over the same lateral range [c1, c2) (positions as in
                                row_col0), the other rows closed; per beam the rectangle with the most negative sum
                                of w; ties: closed aperture at 0, else smallest (c1, c2, m1, m2) */
} dao_mlc_mode;

/* Structures, thresholds and weights of eq. (9)-(10).  One structure per voxel. */
typedef struct {
  int32_t n_struct;              /* <= 255 */
  const int32_t *vox_struct;     /* [n_vox] structure id in [0, n_struct) or -1 (no penalty); same memspace as D */
  const float *t_under;          /* [n_struct] host: T_s^-  (under-dose threshold) */
  const float *w_under;          /* [n_struct] host: alpha_s (0 for non-targets) */
  const float *t_over;           /* [n_struct] host: T_s^+  (over-dose threshold) */
  const float *w_over;           /* [n_struct] host: beta_s */
  /* Re-optimisation mode (the per-voxel form eq. 3-4).  Both fields may be 0. */
  const float *vox_threshold;    /* optional [n_vox], same memspace as D: T_j, replaces BOTH thresholds T_s^- and
                                    T_s^+ of voxel j's structure (finite values) */
  int32_t per_voxel_weights;     /* 0: weights alpha_s / |v_s|, beta_s / |v_s| (eq. 9-10); 1: alpha_s, beta_s are the
                                    per-voxel weights alpha_j, beta_j of eq. 3-4 as they are (no division by |v_s|) */
  /* Voxel-row slab: when D holds only a slab of the voxel rows of a larger problem, |v_s| of eq. 9-10
     is the structure's voxel count in the WHOLE problem, not in the slab.  Optional [n_struct] host array; NULL:
     the context counts its own voxels.  With it, dao_eval_x returns the slab's share of F, dao_spmv_t the slab's
     partial sum of w = D^T pi (eq. 8): the caller adds the shares over the slabs in slab order. */
  const int64_t *struct_count;
} dao_structs;

/* Options.  Zero-initialise, then dao_default_options, then override. */
typedef struct {
  int32_t k_max;             /* capacity of the aperture pool, 1..DAO_MAX_APERTURES (default 50) */
  int32_t master_max_iter;   /* cap on projected-gradient / Newton iterations per master solve (default 2000) */
  double master_tol;         /* stop when max_k |p_k| * max(1, max_k y_k) <= master_tol * F, p = projected
                                steepest-descent direction (default 1e-7); reading S2 */
  double price_tol;          /* optimal iff price_b* >= -price_tol * max_i |w_i| * (rows in b*) (default 1e-6, the
                                fp32 noise floor of w), or iff the best candidate duplicates an aperture of the
                                pool after a CONVERGED master solve whose KKT residual explains the price (the
                                negative price is then residue of that solve); S3, S6 */
  double master_ls_tol;      /* a step t along the search direction is accepted when |phi'(t)| <= master_ls_tol *
                                |phi'(0)| (phi(t) = F(z + t dz)) or when it ends on a bound still descending;
                                otherwise t is refined by a safeguarded Newton search (default 0.01); S2 */
  int32_t master_method;     /* 0 = plain gradient projection, 1 = gradient projection with conjugate
                                (Polak-Ribiere+) directions on the free face, 2 = projected Newton on the free
                                variables (exact Hessian A^T diag(2c) A of the piecewise-quadratic F on the fp64
                                tensor cores, one pass over A per iteration), 3 = the same projected Newton method
                                with the Hessian on the 5th-generation tensor cores (tcgen05, TF32 hi/lo split,
                                TMEM accumulators: H to ~2^-21 relative; dose, objective and gradient -- all
                                that enters the stopping test -- stay fp64; k_max <= 56 only: with a larger
                                pool capacity method 3 runs as method 2); pools of more than 103 apertures
                                use method 1.  dao_get_dims reports the method in effect.  Same stopping test and the same (unique) optimal value for all
                                four; reading S2 */
  int32_t sell_sigma;        /* sorting window (rows) of the internal sliced-ELL layout of D; 1 = keep the
                                caller's voxel order; 0 = library default */
  int32_t timers;            /* non-zero: CUDA-event timers per kernel class in dao_run (default 1) */
  int32_t mlc_mode;          /* dao_mlc_mode (default DAO_MLC_CONSECUTIVE) */
  int32_t reserved;          /* test/bench hooks, 0 in production: bit 0 forces the direct-load SpMV variant,
                                bit 1 turns on the master's phase timers (DAO_VEC_MASTER_PHASES), bit 2 forces the span variant
                                of the transposed SpMV even for short beamlet rows, bit 4 runs the Newton master
                                (methods 2, 3) on 8 CTAs so that small inputs exercise many tiles per CTA */
  int32_t pad_;              /* keep 0 */
} dao_options;

typedef struct {
  size_t workspace_bytes;    /* persistent device memory, lives as long as the context */
  size_t scratch_bytes;      /* device memory needed only during dao_create */
} dao_sizes;

typedef struct {
  int32_t beam;              /* b*: beam of the candidate aperture */
  int32_t converged;         /* 1: no improving aperture exists, no candidate stored */
  double price;              /* reduced cost of the candidate = price_b* (< 0 when it improves) */
  double objective;          /* F(z) at the current intensities */
  double w_abs_max;          /* max_i |w_i| (used by the optimality test) */
  int32_t n_open_beamlets;   /* beamlets opened by the candidate */
  int32_t duplicate;         /* 1: the candidate equals an aperture already in the pool (reading S6) */
  int32_t stalled;           /* 1: the candidate is a duplicate with an improving price after a master solve that did
                                not converge (or whose residue does not explain the price): no candidate is stored and
                                optimality is NOT claimed (converged = 0); solve the master further and price again */
  int32_t reserved;
} dao_price_info;

typedef struct {
  int32_t n_apertures;       /* pool size after the call */
  int32_t n_pg_iter;         /* projected-gradient (methods 0, 1) or Newton (methods 2, 3) iterations taken */
  int32_t hit_max_iter;      /* 1: stopped by master_max_iter */
  int32_t n_restarts;        /* conjugate-direction restarts (method 1) */
  double objective;          /* F(A y) at return */
  double kkt_residual;       /* max_k of |grad_k| where y_k > 0 and max(0, -grad_k) where y_k = 0 */
  double pg_norm;            /* max_k |p_k| at return */
  int32_t n_passes;          /* passes over the aperture-dose block A (4 V K bytes each) */
  int32_t reserved;
} dao_master_info;

typedef struct {
  int32_t n_apertures;
  int32_t n_iterations;      /* column-generation iterations executed by this call */
  int32_t converged;         /* 1: stopped because pricing found no improving aperture */
  int32_t n_duplicates;      /* iterations whose candidate was already in the pool (S6) */
  int64_t n_pg_iter_total;
  double objective;          /* F of the final plan, from the dose SpMV z = D x */
  double seconds_total;      /* device time of the call (CUDA events) */
  /* per kernel class, summed over iterations; zero when options.timers == 0 */
  double seconds_intensity, seconds_spmv, seconds_spmv_t, seconds_price, seconds_column, seconds_master;
  int64_t n_passes_total;    /* passes over the aperture-dose block A made by the master solves of this call */
  int32_t n_hit_max_iter;    /* master solves of this call that stopped on master_max_iter */
  int32_t n_kernel_launches; /* kernels this call launched (counted at the launch sites of the library) */
  int32_t stalled;           /* 1: stopped on a duplicate candidate after an unconverged master solve (S6): converged = 0 */
  int32_t reserved;
} dao_run_info;

/* One record per column-generation iteration, retrievable after dao_run / dao_solve_master. */
typedef struct {
  int32_t k;                 /* pool size after the iteration */
  int32_t beam;
  int32_t n_pg_iter;
  int32_t duplicate;
  double price;
  double objective_before;   /* F before the aperture was added (at pricing time) */
  double objective;          /* F(A y) after the master solve */
  double kkt_residual;
  int32_t n_passes;          /* passes over the aperture-dose block A made by the master solve (4 V K bytes each) */
  int32_t hit_max_iter;      /* 1: that master solve stopped on master_max_iter (or could not make progress) */
} dao_iter_record;

typedef struct {
  int32_t cap_apertures, cap_rows;   /* in: capacities of the arrays below */
  int32_t n_apertures, n_rows_used;  /* out (also set when the capacity is too small -> DAO_E_SHAPE) */
  int32_t *beam;                     /* [cap_apertures] host */
  float *intensity;                  /* [cap_apertures] host, y_k */
  int32_t *ap_row_ptr;               /* [cap_apertures+1] host, into left/right (the rows of that beam, in order) */
  int32_t *left, *right;             /* [cap_rows] host, half-open leaf positions */
  double objective;                  /* F of the plan */
} dao_plan;

typedef enum {               /* dao_get_vector selectors; lengths in elements */
  DAO_VEC_Z = 0,             /* float  [n_vox]  dose of the last evaluation, caller's voxel order */
  DAO_VEC_G = 1,             /* float  [n_vox]  pi_j = dF/dz_j */
  DAO_VEC_W = 2,             /* float  [n_bl]   beamlet gradient */
  DAO_VEC_X = 3,             /* float  [n_bl]   beamlet intensities */
  DAO_VEC_Y = 4,             /* double [k_max]  aperture intensities (first n_apertures valid) */
  DAO_VEC_VSTAR = 5,         /* double [n_rows] row minima of the last pricing */
  DAO_VEC_LEFT = 6,          /* int32  [n_rows] */
  DAO_VEC_RIGHT = 7,         /* int32  [n_rows] */
  DAO_VEC_BEAM_PRICE = 8,    /* double [n_beams] */
  DAO_VEC_HISTORY = 9,       /* dao_iter_record [k_max] (first n_apertures valid) */
  DAO_VEC_MASTER_Z = 10,     /* double [n_vox]  z = A y as the master holds it, caller's voxel order */
  DAO_VEC_ITER_SECONDS = 12, /* double [k_max][6]  HOST only: one row per aperture the last dao_run ADDED, in order (row i
                                belongs to the i-th history record that call wrote): device seconds per kernel class
                                {intensity, dose SpMV, SpMV^T, pricing, column, master} of the iteration that added it,
                                plus those of preceding iterations that added nothing (a stalled pricing and its master
                                re-solve, S6).  The last pricing of a run that ends converged or stalled adds no row; its
                                time is in dao_run_info.seconds_*.  CUDA events; zeros when options.timers == 0 and
                                beyond the rows written */
  DAO_VEC_MASTER_PHASES = 11 /* uint64 [16]     phase timers of the master kernel, accumulated since dao_create when
                                dao_options.reserved has bit 1 (value 2) set, else zeros.  Nanoseconds of CTA 0 in:
                                0 set-up and z = A y, 1 gradient pass over A, 2 gradient reduction, 3 direction,
                                4 dz = A p pass, 5 curvature reduction, 6 line search, 10 publish, 14 accept / refine decision (split off
                                slot 3); counts:
                                7 line-search evaluations, 8 projected-gradient iterations, 9 calls; SM clock cycles thread 0 of
                                CTA 0 spent waiting for stages of A: 12 in gradient passes, 13 in dz passes */
} dao_vector;

void dao_default_options(dao_options *opt);

/* Sizes of the two device buffers dao_create needs for this problem.  Reads D->row_ptr. */
dao_status dao_workspace_bytes(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s,
                               const dao_options *opt, dao_sizes *out);

/* Validate the inputs, copy them to the device, build the internal layouts (sliced-ELL of D, CSR
 * of D^T, pricing tables, per-structure penalty table) inside `workspace`, and start with an empty
 * aperture pool (z = 0).  Both buffers must be 256-byte aligned device memory of at least the
 * sizes dao_workspace_bytes reported; `scratch` may be released when the call returns.
 * cuda_stream is a cudaStream_t (NULL = legacy default stream).  On failure *out = NULL and the
 * message is available from dao_last_error(NULL). */
dao_status dao_create(const dao_csr *D, const dao_mlc *mlc, const dao_structs *s, const dao_options *opt,
                      void *workspace, size_t workspace_bytes, void *scratch, size_t scratch_bytes,
                      void *cuda_stream, dao_ctx **out);

/* Steps 1-6 at the current intensities.  Stores the candidate aperture; the pool is unchanged. */
dao_status dao_price(dao_ctx *ctx, dao_price_info *out);

/* Steps 7-8: append the pending candidate (DAO_E_STATE if there is none or the pool is full), then
 * solve the restricted master problem over the pool on the device. */
dao_status dao_solve_master(dao_ctx *ctx, dao_master_info *out);

/* Step 9: repeat price -> add -> master until the pool holds max_apertures apertures or pricing
 * proves optimality.  One host synchronisation per iteration.  Ends with a final dose evaluation
 * (steps 1-3) so that DAO_VEC_Z / objective describe the returned plan. */
dao_status dao_run(dao_ctx *ctx, int32_t max_apertures, dao_run_info *out);

/* Copy the plan into caller-allocated host arrays. */
dao_status dao_get_plan(dao_ctx *ctx, dao_plan *out);

/* Empty the pool (y, z back to the state after dao_create); keeps the matrix layouts. */
dao_status dao_reset(dao_ctx *ctx);

dao_status dao_destroy(dao_ctx *ctx);

/* Message of the last failure of this context (ctx = NULL: of the last failed dao_create /
 * dao_workspace_bytes on this thread).  Owned by the library, valid until the next call. */
const char *dao_last_error(const dao_ctx *ctx);

/* ---- test / bench hooks (parity harness, BASELINE.json configs[3] kernel sweep) ---------------- */

/* Copy an internal vector to `dst` (host or device memory, see dao_vector for type and length). */
dao_status dao_get_vector(dao_ctx *ctx, int32_t which, void *dst, dao_memspace mem);

/* Problem dimensions and layout facts. */
typedef struct {
  int32_t n_vox, n_bl, n_beams, n_rows, n_struct, k_max;
  int64_t nnz;               /* of D as given */
  int64_t sell_elems;        /* stored elements of the sliced-ELL copy (>= nnz: padding) */
  int32_t sell_slice_rows, sell_sigma;
  int32_t n_sm;
  int32_t master_method;     /* the master method in effect (dao_options.master_method after the capacity fallbacks) */
} dao_dims;
dao_status dao_get_dims(const dao_ctx *ctx, dao_dims *out);

/* Isolated kernels on caller-provided DEVICE vectors in the caller's voxel / beamlet order.
 * Asynchronous on the context's stream (no synchronisation). */
dao_status dao_spmv(dao_ctx *ctx, const float *x_dev, float *z_dev);        /* z = D x        [n_bl] -> [n_vox] */
dao_status dao_spmv_t(dao_ctx *ctx, const float *g_dev, float *w_dev);      /* w = D^T g      [n_vox] -> [n_bl] */
/* Dose + objective + gradient for given beamlet intensities: steps 2-3.  Synchronises. */
dao_status dao_eval_x(dao_ctx *ctx, const float *x_dev, double *objective);
/* Steps 5-6 on a caller-provided fp32 beamlet-gradient vector (DEVICE, [n_bl]) and caller-provided
 * MLC tables (DEVICE, n_rows+1 / n_beams+1 entries; pass NULL, NULL, 0, 0 to use the context's).
 * Outputs are DEVICE arrays: left/right int32 [n_rows], vstar double [n_rows], beam_price double
 * [n_beams], best int32 [1].  Asynchronous. */
dao_status dao_price_from_w(dao_ctx *ctx, const float *w_dev, const int32_t *row_bl_ptr_dev,
                            const int32_t *beam_row_ptr_dev, int32_t n_rows, int32_t n_beams,
                            int32_t *left_dev, int32_t *right_dev, double *vstar_dev,
                            double *beam_price_dev, int32_t *best_dev);
/* ---- pricing for callers that cannot allocate device memory ---------------------------------------
 * Steps 5-6 (per leaf row the most negative contiguous interval, per-beam sums, best beam)
 * with NO context, NO workspace and NO allocation of any kind: the same row kernel and the same last-CTA tail
 * as dao_price_from_w, but the intermediate arrays the tail needs (max |w| per leaf row and per beam, the
 * ticket counter that elects the last CTA) live in a fixed array compiled into the library image instead of in
 * a dao_create workspace.
 *
 * Who this is for.  Every other call of this library works inside a context, and a context needs a workspace
 * somebody obtained from cudaMalloc (or from a framework's allocator, which calls it).  Some hosts of a pricing
 * step cannot do that at the moment they need the answer: a treatment-console process whose device memory was
 * handed out in full at start-up and is owned by another component; a plug-in that is given device pointers by
 * its host application but no allocator; a delivery-time safety loop whose coding rules forbid any call that
 * may block on the driver's allocator lock or grow the process footprint (cudaMalloc and cudaFree both
 * synchronise the device and can fail late, when there is nobody left to handle it).  Such a caller already
 * owns w and the MLC tables and somewhere to put the answer; this entry point asks for nothing else.
 *
 * Arguments: as dao_price_from_w with caller tables -- all DEVICE pointers on the CURRENT device, which must
 * also be the device of `cuda_stream` (NULL = legacy default stream): w_dev fp32 [row_bl_ptr[n_rows]];
 * row_bl_ptr_dev int32 [n_rows+1] and beam_row_ptr_dev int32 [n_beams+1], both starting at 0 and non-decreasing
 * (not checked: they are device data); outputs left/right int32 [n_rows] (half-open leaves inside the row,
 * closed row = (0, 0)), vstar double [n_rows], beam_price double [n_beams], best int32 [1].  Consecutive-leaf
 * rule only (DAO_MLC_CONSECUTIVE).  Asynchronous: nothing is synchronised; outputs are valid once the stream
 * reaches the end of the launch.  Bit-identical to dao_price_from_w on the same inputs.
 *
 * Limits.  1 <= n_rows <= DAO_STATIC_MAX_ROWS and 1 <= n_beams <= DAO_STATIC_MAX_BEAMS, otherwise DAO_E_SHAPE
 * with the limit named in dao_last_error(NULL) and nothing launched.  The fixed array is DAO_STATIC_SCRATCH_BYTES
 * (136 KiB) of device memory on every GPU that loads the library, held until the process exits, whether or not
 * this function is ever called.
 *
 * First call on a device: the library looks up the array's device address (cudaGetSymbolAddress, once per
 * device, with that device current; this is also what makes the CUDA runtime load the library's device code
 * if nothing has yet).  Make that first call during start-up, outside any stream capture and before timing
 * matters; later calls on that device only enqueue a 256-byte memset of the ticket and one kernel.
 *
 * Sharing.  All calls on a device use the one array, and it keeps whatever the previous call left there.  The
 * function clears the part that must start at zero (the ticket) in stream order before its kernel; the rest is
 * fully rewritten before it is read.  Two calls whose kernels can overlap on the GPU (different streams, or
 * different host threads on different streams) RACE on it and return garbage: issue them on one stream, or
 * order them with events.  Calls from several host threads on the same stream are safe. */
#define DAO_STATIC_MAX_ROWS 16384
#define DAO_STATIC_MAX_BEAMS 1024
#define DAO_STATIC_SCRATCH_BYTES (256 + 8 * DAO_STATIC_MAX_ROWS + 8 * DAO_STATIC_MAX_BEAMS)
dao_status dao_price_from_w_static(const float *w_dev, const int32_t *row_bl_ptr_dev,
                                   const int32_t *beam_row_ptr_dev, int32_t n_rows, int32_t n_beams,
                                   int32_t *left_dev, int32_t *right_dev, double *vstar_dev,
                                   double *beam_price_dev, int32_t *best_dev, void *cuda_stream);

/* Load a pool of apertures (host arrays laid out as in dao_plan) with intensities y (host, may be
 * NULL = zeros) replacing the current pool: builds the dose columns (step 7) but does not solve.
 * Lets the parity harness solve the master on the oracle's pool. */
dao_status dao_set_pool(dao_ctx *ctx, int32_t n_apertures, const int32_t *beam, const int32_t *ap_row_ptr,
                        const int32_t *left, const int32_t *right, const double *y);
/* Solve the restricted master over the current pool without adding a column. */
dao_status dao_resolve_master(dao_ctx *ctx, dao_master_info *out);

/* ---- FMO workload ------------------------------------------------------------------
 * Fluence-map optimisation: the same objective with the beamlet intensities as the decision
 * variables, min_{x >= 0} F(D x).  "Mathematically, the DAO model is the same as the FMO model ...
 * in which the decision variables are the intensities of all beamlets", solved by "the same gradient
 * projection method".  By eq. (7) its optimum is a lower bound
 * of every aperture plan's objective.  Runs steps 2-4 of the hot path (dose SpMV + fused objective /
 * gradient, transposed SpMV) plus a projected-gradient update per iteration, entirely on the device;
 * the host reads a small state block every `check_every` iterations. */
typedef struct {
  int32_t n_iter;            /* projected-gradient iterations done */
  int32_t converged;         /* 2: F stopped decreasing beyond fp64 rounding (resolution of the fp32 gradient);
                                1: max_i |x_i - max(0, x_i - t w_i)| / t * max(1, max x) <= tol * F, t = last step */
  int32_t hit_max_iter;
  int32_t n_restarts;        /* steepest-descent restarts of the conjugated direction */
  int32_t n_ls_evals;        /* line-search evaluations of phi'(t) (passes over z, dz only) */
  int32_t reserved;
  double objective;          /* F(D x) at the returned x */
  double kkt_residual;       /* that measure over x_i > 0, and max(0, -w_i) where x_i = 0 */
  double pg_norm;            /* max_i |p_i| of the projected steepest-descent direction */
  double seconds;            /* device time of the solve */
} dao_fmo_info;
/* Solve from x = 0 (warm_start = 0) or from the context's current DAO_VEC_X (warm_start = 1).
 * tol <= 0 selects dao_options.master_tol; the conjugation follows dao_options.master_method.  On
 * return DAO_VEC_X / DAO_VEC_Z / DAO_VEC_G / DAO_VEC_W describe the returned x.  The aperture pool of
 * the context is not touched, but its last dose evaluation is overwritten. */
dao_status dao_fmo_solve(dao_ctx *ctx, int32_t max_iter, double tol, int32_t warm_start, dao_fmo_info *out);

#ifdef __cplusplus
}
#endif
#endif /* DAO_H_ */
