// dao_pricing.cu -- the pricing sub-problem, PAPER.md:136-169 (eq. 8):
//   step 5  per MLC leaf row the contiguous interval with the most negative sum of w
//   step 6  per-beam sum of the row minima, beam with the smallest sum, optimality test,
//           and the bookkeeping that turns the winner into the pending candidate aperture.
#include "dao_internal.cuh"

#include <math_constants.h>

#include <algorithm>
#include <mutex>
#include <string>

namespace dao {

constexpr int kPriceSeqMaxLen = 88;    // longest leaf row the thread-per-row kernel stages
constexpr int kPriceSeqMinRows = 32768; // below this the warp-per-row kernel has the lower latency

// The tail of a pricing launch: the LAST CTA to finish (ticket counter) sums the row minima per beam (step 6a),
// picks the beam, tests optimality and, inside dao_run / dao_price, turns the winner into the pending candidate
// (pool tables at index K, 0/1 beamlet mask) -- one launch instead of four (row kernel, beam sums, selection,
// append).  Every kernel that ends with it runs 256 threads per CTA and no thread leaves before the tail.
struct PriceTail {
  uint32_t *ticket;              // self-resetting counter (DevState.ticket_misc: free between the SpMV^T and the column)
  int32_t do_beams;              // 1: the kernel produced row minima, the beam sums are still to do
  int32_t n_beams, n_rows, n_bl, max_rows, k_max;
  const int32_t *beam_row_ptr, *row_bl_ptr, *bl_row, *row_beam;
  double *vstar, *row_absmax, *beam_price, *beam_absmax;
  int32_t *left, *right, *best_out;
  DevState *st;                  // null: hook call (dao_price_from_w), no candidate bookkeeping
  double price_tol;
  int32_t *ap_beam, *ap_left, *ap_right;
  unsigned long long *ap_hash;
  float *xmask;
};
__device__ void price_tail(const PriceTail &q);

// ------------------------------------------------------------------------------------------
// step 5.  One warp per leaf row.  With S_0 = 0 and S_r = w_1 + .. + w_r (fp64 sums of the fp32
// inputs) the printed scan returns
//     v* = min_r ( S_r - max_{0<=l<=r} S_l ),   l = first index attaining the prefix maximum,
// taking the first r that attains the minimum; the closed row wins every tie at 0.  This equals
// the lexicographically smallest (value, l, r) over all intervals (reading S4).
// The warp does an inclusive sum scan, an inclusive (max, first-argmax) scan and an argmin
// reduction per tile of 32 beamlets, carrying (S, max, argmax, best) between tiles.
// Output in the ABI convention: half-open [left, right) = [l, r), closed row = (0, 0).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void price_rows_body(const float *__restrict__ w, const int32_t *__restrict__ row_bl_ptr,
                                                int32_t n_rows, double *__restrict__ vstar, int32_t *__restrict__ left,
                                                int32_t *__restrict__ right, double *__restrict__ row_absmax,
                                                const int32_t *__restrict__ maxlen_flag) {
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (maxlen_flag && *maxlen_flag <= kPriceSeqMaxLen) return;     // the thread-per-row kernel takes this launch
  if (row >= n_rows) return;
  const int32_t b0 = row_bl_ptr[row];
  const int32_t n = row_bl_ptr[row + 1] - b0;
  const unsigned FULL = 0xffffffffu;

  double carry = 0.0;                  // S at the end of the previous tile
  double run_max = 0.0;                // max_{0<=l<=r} S_l so far (S_0 = 0 at l = 0)
  int32_t run_arg = 0;
  double best = 0.0;                   // v*
  int32_t best_l = 0, best_r = 0;      // closed
  double amax = 0.0;

  for (int32_t base = 0; base < n; base += 32) {
    const int32_t idx = base + lane;
    const bool valid = idx < n;
    const double wv = valid ? (double)w[b0 + idx] : 0.0;
    amax = fmax(amax, fabs(wv));
    // inclusive prefix sum
    double s = wv;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double t = __shfl_up_sync(FULL, s, o);
      if (lane >= o) s += t;
    }
    const double P = carry + s;        // S_r with r = idx + 1
    // inclusive prefix (max, first argmax)
    double mv = valid ? P : -CUDART_INF;
    int32_t mi = idx + 1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double tv = __shfl_up_sync(FULL, mv, o);
      const int32_t ti = __shfl_up_sync(FULL, mi, o);
      if (lane >= o && tv >= mv) { mv = tv; mi = ti; }   // ties keep the smaller index
    }
    if (run_max >= mv) { mv = run_max; mi = run_arg; }
    // candidate of this r: value, l, r
    double cv = valid ? (P - mv) : 0.0;
    int32_t cl = mi, cr = idx + 1;
    if (!(cv < 0.0)) { cv = 0.0; cl = 0; cr = 0; }        // never open a non-improving interval
    // lexicographic argmin over the tile
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(FULL, cv, o);
      const int32_t ol = __shfl_xor_sync(FULL, cl, o);
      const int32_t orr = __shfl_xor_sync(FULL, cr, o);
      const bool take = (ov < cv) || (ov == cv && (ol < cl || (ol == cl && orr < cr)));
      if (take) { cv = ov; cl = ol; cr = orr; }
    }
    if ((cv < best) || (cv == best && cv < 0.0 && (cl < best_l || (cl == best_l && cr < best_r)))) {
      best = cv; best_l = cl; best_r = cr;
    }
    carry += __shfl_sync(FULL, s, 31);
    run_max = __shfl_sync(FULL, mv, 31);
    run_arg = __shfl_sync(FULL, mi, 31);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmax(amax, __shfl_xor_sync(FULL, amax, o));
  if (lane == 0) {
    vstar[row] = best;
    left[row] = best_l;
    right[row] = best_r;
    row_absmax[row] = amax;
  }
}

__global__ void __launch_bounds__(256) k_price_rows(const float *w, const int32_t *row_bl_ptr, int32_t n_rows, double *vstar,
                                                    int32_t *left, int32_t *right, double *row_absmax,
                                                    const int32_t *maxlen_flag, PriceTail tail) {
  price_rows_body(w, row_bl_ptr, n_rows, vstar, left, right, row_absmax, maxlen_flag);
  if (tail.ticket) price_tail(tail);
}

// ------------------------------------------------------------------------------------------
// step 5 for MANY leaf rows (the 10^4-10^5-row end of BASELINE.json configs[3]): thread per row, which is the
// paper's own launch shape, but fed through shared memory: a warp copies the beamlets of its 32
// consecutive rows (one contiguous slice of w) with coalesced loads, then every lane runs the printed scan
// over its own row sequentially in fp64 -- the paper's loop as printed, strict comparisons
// included, so ties and sums agree bit for bit.  The warp-per-row kernel above stays in use for few rows
// (lower latency) and for rows too long for the staging buffer.
// ------------------------------------------------------------------------------------------
constexpr int kPriceStageFloats = 33 * kPriceSeqMaxLen;    // per warp: 32 rows of up to 88 beamlets + 1 word of skew per 32 (46.5 KB static per CTA) (+ skew against bank conflicts)
__global__ void __launch_bounds__(128) k_price_rows_seq(const float *__restrict__ w,
                                                        const int32_t *__restrict__ row_bl_ptr, int32_t n_rows,
                                                        double *__restrict__ vstar, int32_t *__restrict__ left,
                                                        int32_t *__restrict__ right, double *__restrict__ row_absmax,
                                                        const int32_t *__restrict__ maxlen_flag) {
  __shared__ float stage[4][kPriceStageFloats];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (maxlen_flag && *maxlen_flag > kPriceSeqMaxLen) return;      // rows too long: the warp-per-row kernel runs
  const int row0 = (blockIdx.x * 4 + warp) * 32;
  if (row0 >= n_rows) return;
  const int rows = min(32, n_rows - row0);
  const int32_t b0 = row_bl_ptr[row0], b1 = row_bl_ptr[row0 + rows];
  float *buf = stage[warp];
  // element e of the slice goes to buf[e + e / 32]: consecutive rows start 1 word further apart than their
  // length, which spreads the lanes' sequential reads over the banks for the usual equal-length rows
  for (int32_t e = lane; e < b1 - b0; e += 32) buf[e + (e >> 5)] = w[b0 + e];
  __syncwarp();
  if (lane >= rows) return;
  const int row = row0 + lane;
  const int32_t s0 = row_bl_ptr[row] - b0, n = row_bl_ptr[row + 1] - row_bl_ptr[row];
  double v = 0.0, vbar = 0.0, best = 0.0, amax = 0.0;
  int32_t l = 0, bl = 0, br = 0;
  for (int32_t i = 0; i < n; ++i) {
    const int32_t e = s0 + i;
    const double wv = (double)buf[e + (e >> 5)];
    amax = fmax(amax, fabs(wv));
    v += wv;
    if (v > vbar) { vbar = v; l = i + 1; }            // :163
    if (v - vbar < best) { best = v - vbar; bl = l; br = i + 1; }   // :165
  }
  vstar[row] = best; left[row] = bl; right[row] = br; row_absmax[row] = amax;
}

// longest leaf row of device-resident MLC tables (the caller's, in dao_price_from_w)
__global__ void k_price_maxlen(const int32_t *__restrict__ row_bl_ptr, int32_t n_rows, int32_t *__restrict__ out) {
  int m = 0;
  for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < n_rows; r += gridDim.x * blockDim.x)
    m = max(m, row_bl_ptr[r + 1] - row_bl_ptr[r]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// step 6a: price_b = sum over the rows of beam b of v* (PAPER.md:169).  One warp per beam,
// lane-strided partial sums in row order, then a fixed shuffle tree.
__device__ __forceinline__ void price_beam_body(int b, const double *vstar, const double *row_absmax,
                                                const int32_t *__restrict__ beam_row_ptr, double *beam_price,
                                                double *beam_absmax) {
  const int lane = threadIdx.x & 31;
  double s = 0.0, a = 0.0;
  for (int32_t r = beam_row_ptr[b] + lane; r < beam_row_ptr[b + 1]; r += 32) {
    s += __ldcg(vstar + r);
    a = fmax(a, __ldcg(row_absmax + r));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s += __shfl_xor_sync(0xffffffffu, s, o);
    a = fmax(a, __shfl_xor_sync(0xffffffffu, a, o));
  }
  if (lane == 0) {
    beam_price[b] = s;
    beam_absmax[b] = a;
  }
}

__global__ void __launch_bounds__(256) k_price_beams(const double *vstar, const double *row_absmax,
                                                     const int32_t *beam_row_ptr, int32_t n_beams, double *beam_price,
                                                     double *beam_absmax) {
  const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (b < n_beams) price_beam_body(b, vstar, row_absmax, beam_row_ptr, beam_price, beam_absmax);
}

// ------------------------------------------------------------------------------------------
// Jaws-only pricing (PAPER.md:260 names the constraint; reading J1 of DESIGN.md): per beam the rectangle
// (consecutive leaf rows m1..m2, one common lateral range [c1, c2)) with the most negative sum of w.
// One CTA per beam.  Prefix sums of every row over lateral positions (fp64, zero where the row has no
// beamlet) go to shared memory; every thread takes column pairs (c1, c2) in ascending order and runs the
// paper's one-pass scan over the ROWS on the row sums P[m][c2] - P[m][c1]; a block
// argmin with the key (value, c1, c2) picks the winner.  Strict comparisons everywhere: the closed aperture
// wins ties at 0, equal negative values keep the smallest (c1, c2, m1, m2) -- the oracle's enumeration order.
// Outputs per row: the rectangle clipped to the row's beamlets as half-open leaves inside the row, and the
// sum of w over them.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void price_jaws_body(const float *__restrict__ w, const int32_t *__restrict__ beam_row_ptr,
                                                    const int32_t *__restrict__ row_bl_ptr,
                                                    const int32_t *__restrict__ row_col0, int32_t width,
                                                    double *__restrict__ vstar, int32_t *__restrict__ left,
                                                    int32_t *__restrict__ right, double *__restrict__ beam_price,
                                                    double *__restrict__ beam_absmax) {
  extern __shared__ double P[];                     // [R][width + 1]
  __shared__ double s_val[256];
  __shared__ int32_t s_c1[256], s_c2[256], s_m1[256], s_m2[256];
  __shared__ double s_abs[256];
  const int t = threadIdx.x, b = blockIdx.x;
  const int32_t r0 = beam_row_ptr[b], R = beam_row_ptr[b + 1] - r0;
  const int ld = width + 1;
  double amax = 0.0;
  for (int m = t; m < R; m += 256) {                // one thread per row: sequential prefix sum, left to right
    const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, b0 = row_bl_ptr[r], n = row_bl_ptr[r + 1] - b0;
    double s = 0.0;
    P[m * ld] = 0.0;
    for (int c = 0; c < width; ++c) {
      if (c >= c0 && c < c0 + n) {
        const double wv = (double)w[b0 + (c - c0)];
        s += wv;
        amax = fmax(amax, fabs(wv));
      }
      P[m * ld + c + 1] = s;
    }
  }
  __syncthreads();
  double best = 0.0;
  int32_t bc1 = 0, bc2 = 0, bm1 = 0, bm2 = 0;       // closed: m2 exclusive, empty range
  for (int c1 = 0; c1 < width; ++c1) {
    for (int c2 = c1 + 1 + t; c2 <= width; c2 += 256) {
      double v = 0.0, vbar = 0.0;
      int32_t l = 0;
      for (int m = 0; m < R; ++m) {
        v += P[m * ld + c2] - P[m * ld + c1];
        if (v - vbar < best) { best = v - vbar; bc1 = c1; bc2 = c2; bm1 = l; bm2 = m + 1; }
        if (v > vbar) { vbar = v; l = m + 1; }
      }
    }
  }
  s_val[t] = best; s_c1[t] = bc1; s_c2[t] = bc2; s_m1[t] = bm1; s_m2[t] = bm2; s_abs[t] = amax;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (t < o) {
      const double ov = s_val[t + o];
      const bool take = ov < s_val[t] ||
                        (ov == s_val[t] && ov < 0.0 &&
                         (s_c1[t + o] < s_c1[t] || (s_c1[t + o] == s_c1[t] && s_c2[t + o] < s_c2[t])));
      if (take) { s_val[t] = ov; s_c1[t] = s_c1[t + o]; s_c2[t] = s_c2[t + o]; s_m1[t] = s_m1[t + o]; s_m2[t] = s_m2[t + o]; }
      s_abs[t] = fmax(s_abs[t], s_abs[t + o]);
    }
    __syncthreads();
  }
  const int32_t c1 = s_c1[0], c2 = s_c2[0], m1 = s_m1[0], m2 = s_m2[0];
  for (int m = t; m < R; m += 256) {
    const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, n = row_bl_ptr[r + 1] - row_bl_ptr[r];
    int32_t lo = max(c1, c0), hi = min(c2, c0 + n);
    if (m < m1 || m >= m2 || hi <= lo) { lo = c0; hi = c0; }
    left[r] = hi > lo ? lo - c0 : 0;
    right[r] = hi > lo ? hi - c0 : 0;
    vstar[r] = P[m * ld + hi] - P[m * ld + lo];
  }
  if (t == 0) {
    beam_price[b] = s_val[0];
    beam_absmax[b] = s_abs[0];
  }
}

__global__ void __launch_bounds__(256) k_price_jaws(const float *w, const int32_t *beam_row_ptr, const int32_t *row_bl_ptr,
                                                    const int32_t *row_col0, int32_t width, double *vstar, int32_t *left,
                                                    int32_t *right, double *beam_price, double *beam_absmax,
                                                    PriceTail tail) {
  price_jaws_body(w, beam_row_ptr, row_bl_ptr, row_col0, width, vstar, left, right, beam_price, beam_absmax);
  if (tail.ticket) price_tail(tail);
}

// ------------------------------------------------------------------------------------------
// Interdigitation (reading J2) and connectedness (reading J3) pricing (PAPER.md:260 names the constraints):
// the feasible apertures of a beam are chains over its leaf rows, so the best one is a shortest path through
// the layered graph rows x leaf states (a, b) (lateral tip positions, 0 <= a <= b <= W; closed when a == b):
//   f_m(s) = val_m(s) + min { f_{m-1}(s') : s' compatible with s }.
// One CTA per beam; the row prefix sums and two layers of f live in shared memory, the back-pointers in the
// workspace.  Both compatibility rules are dominance conditions (a' <= x, b' >= y), so the inner minimum is a
// 2-D prefix minimum of the previous layer: two sweeps of O(W^2) per row instead of O(W^4) comparisons, with the
// key (value, state index), which reproduces the oracle's choice (first minimiser in state order) among equal
// minima.  Thread 0 walks the back-pointers.
//   J2: a_m <= b_{m+1} and a_{m+1} <= b_m for adjacent rows (a closed pair may park anywhere in [0, W]);
//   J3: the open rows are consecutive and adjacent open intervals share a lateral position.
// An open row stays inside its own beamlets.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void price_chain_body(int32_t mode, const float *__restrict__ w,
                                                     const int32_t *__restrict__ beam_row_ptr,
                                                     const int32_t *__restrict__ row_bl_ptr,
                                                     const int32_t *__restrict__ row_col0, int32_t width, int32_t max_rows,
                                                     int32_t *__restrict__ from_g /* [n_rows][(width+1)^2] */,
                                                     double *__restrict__ vstar, int32_t *__restrict__ left,
                                                     int32_t *__restrict__ right, double *__restrict__ beam_price,
                                                     double *__restrict__ beam_absmax) {
  extern __shared__ double sm_d[];
  const int ld = width + 1, S = ld * ld;                    // state (a, b) has index a * ld + b (valid when a <= b)
  double *P = sm_d;                                         // [max_rows][ld] row prefix sums over lateral positions
  double *fp = P + (size_t)max_rows * ld;                   // [S] previous layer (inf = infeasible)
  double *fc = fp + S;                                      // [S] current layer
  double *G = fc + S;                                       // [S] G[x][y] = min { f_prev(a', b') : a' <= x, b' >= y }
  int32_t *Garg = reinterpret_cast<int32_t *>(G + S);       // [S] its first minimiser in state order
  __shared__ double s_val[256];
  __shared__ int32_t s_m[256], s_s[256];
  __shared__ double s_abs[256];
  const int t = threadIdx.x, b = blockIdx.x;
  const int32_t r0 = beam_row_ptr[b], R = beam_row_ptr[b + 1] - r0;
  if (R == 0) {                                             // a beam without leaf rows: only the closed aperture
    if (t == 0) { beam_price[b] = 0.0; beam_absmax[b] = 0.0; }
    return;
  }
  double amax = 0.0;
  for (int m = t; m < R; m += 256) {
    const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, b0 = row_bl_ptr[r], n = row_bl_ptr[r + 1] - b0;
    double s = 0.0;
    P[m * ld] = 0.0;
    for (int c = 0; c < width; ++c) {
      if (c >= c0 && c < c0 + n) {
        const double wv = (double)w[b0 + (c - c0)];
        s += wv;
        amax = fmax(amax, fabs(wv));
      }
      P[m * ld + c + 1] = s;
    }
  }
  __syncthreads();
  double best = (mode == 3) ? 0.0 : CUDART_INF;            // J3: best end of an open run seen by this thread
  int32_t best_m = -1, best_s = -1;
  for (int m = 0; m < R; ++m) {
    const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, n = row_bl_ptr[r + 1] - row_bl_ptr[r];
    if (m > 0) {
      // 2-D prefix minimum of the previous layer with the key (value, state index): first along a' ...
      for (int y = t; y < ld; y += 256) {
        double v = CUDART_INF;
        int32_t arg = -1;
        for (int x = 0; x < ld; ++x) {
          const double f = fp[x * ld + y];
          if (f < v) { v = f; arg = x * ld + y; }           // ascending a': ties keep the smaller index
          G[x * ld + y] = v;
          Garg[x * ld + y] = arg;
        }
      }
      __syncthreads();
      // ... then along b' (descending), comparing indices on ties
      for (int x = t; x < ld; x += 256) {
        double v = CUDART_INF;
        int32_t arg = -1;
        for (int y = ld - 1; y >= 0; --y) {
          const double f = G[x * ld + y];
          const int32_t fa = Garg[x * ld + y];
          if (fa >= 0 && (f < v || (f == v && fa < arg))) { v = f; arg = fa; }
          G[x * ld + y] = v;
          Garg[x * ld + y] = arg;
        }
      }
      __syncthreads();
    }
    int32_t *from = from_g + (size_t)(r0 + m) * S;
    for (int s = t; s < S; s += 256) {
      const int a = s / ld, bb = s - a * ld;
      double out = CUDART_INF;
      int32_t arg = -1;
      const bool open = a < bb;
      const bool valid = a <= bb && (open ? (a >= c0 && bb <= c0 + n) : (mode != 3));
      if (valid) {
        const double val = open ? P[m * ld + bb] - P[m * ld + a] : 0.0;
        double prev = 0.0;
        bool ok = true;
        if (m > 0) {
          if (mode == 2) {                                  // a' <= b and b' >= a
            prev = G[bb * ld + a];
            arg = Garg[bb * ld + a];
            ok = arg >= 0;
          } else {                                          // overlap: a' <= b - 1 and b' >= a + 1; or start the run here
            const double gv = G[(bb - 1) * ld + (a + 1)];
            if (gv < 0.0) { prev = gv; arg = Garg[(bb - 1) * ld + (a + 1)]; }
          }
        }
        if (ok) {
          out = val + prev;
          if (mode == 3 && out < best) { best = out; best_m = m; best_s = s; }
        }
      }
      fc[s] = out;
      from[s] = arg;
    }
    __syncthreads();
    double *tmp = fp; fp = fc; fc = tmp;
  }
  if (mode == 2) {                                          // best state of the last row (fp = last layer)
    best = CUDART_INF; best_m = R - 1; best_s = -1;
    for (int s = t; s < S; s += 256)
      if (fp[s] < best) { best = fp[s]; best_s = s; }
  }
  s_val[t] = best; s_m[t] = best_m; s_s[t] = best_s; s_abs[t] = amax;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (t < o) {
      const double ov = s_val[t + o];
      const int om = s_m[t + o], os = s_s[t + o];
      // key (value, m, s); an entry without a state (s < 0) only carries the neutral value
      const bool take = os >= 0 && (s_s[t] < 0 || ov < s_val[t] ||
                                    (ov == s_val[t] && (om < s_m[t] || (om == s_m[t] && os < s_s[t]))));
      if (take) { s_val[t] = ov; s_m[t] = om; s_s[t] = os; }
      s_abs[t] = fmax(s_abs[t], s_abs[t + o]);
    }
    __syncthreads();
  }
  for (int m = t; m < R; m += 256) { left[r0 + m] = 0; right[r0 + m] = 0; vstar[r0 + m] = 0.0; }
  __threadfence_block();
  __syncthreads();
  if (t == 0) {
    double price = s_val[0];
    int m = s_m[0], s = s_s[0];
    if (s < 0) { price = 0.0; m = -1; }                     // nothing improves: closed aperture
    for (; m >= 0 && s >= 0; --m) {
      const int a = s / ld, bb = s - a * ld;
      if (a < bb) {
        const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0;
        left[r] = a - c0; right[r] = bb - c0;
        vstar[r] = P[m * ld + bb] - P[m * ld + a];
      }
      s = from_g[(size_t)(r0 + m) * S + s];
    }
    beam_price[b] = price;
    beam_absmax[b] = s_abs[0];
  }
}

__global__ void __launch_bounds__(256) k_price_chain(int32_t mode, const float *w, const int32_t *beam_row_ptr,
                                                     const int32_t *row_bl_ptr, const int32_t *row_col0, int32_t width,
                                                     int32_t max_rows, int32_t *from_g, double *vstar, int32_t *left,
                                                     int32_t *right, double *beam_price, double *beam_absmax,
                                                     PriceTail tail) {
  price_chain_body(mode, w, beam_row_ptr, row_bl_ptr, row_col0, width, max_rows, from_g, vstar, left, right, beam_price,
                   beam_absmax);
  if (tail.ticket) price_tail(tail);
}

// step 6b: b* = argmin_b price_b (ties: smallest b), optimality test (reading S3), candidate
// bookkeeping.  One CTA.
// (a device function run by one CTA of 256 threads: the tail of the pricing launch, or k_price_select; what other
// CTAs of the same launch wrote is read with __ldcg)
__device__ void price_select_body(const double *beam_price, const double *beam_absmax, int32_t n_beams,
                                  const int32_t *__restrict__ beam_row_ptr, const int32_t *left, const int32_t *right,
                                  int32_t *best_out, DevState *st, double price_tol, int32_t k_max, int32_t max_rows,
                                  const int32_t *ap_beam, const int32_t *ap_left, const int32_t *ap_right,
                                  const unsigned long long *ap_hash) {
  __shared__ double sv[256];
  __shared__ int32_t sb[256];
  __shared__ double sa[256];
  __shared__ int32_t s_cnt[256];
  const int t = threadIdx.x;
  double bv = CUDART_INF, am = 0.0;
  int32_t bb = 0x7fffffff;
  for (int32_t b = t; b < n_beams; b += 256) {
    const double v = __ldcg(beam_price + b);
    if (v < bv) { bv = v; bb = b; }     // ascending b within a thread: ties keep the smaller b
    am = fmax(am, __ldcg(beam_absmax + b));
  }
  sv[t] = bv; sb[t] = bb; sa[t] = am;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (t < o) {
      const double ov = sv[t + o];
      const int32_t ob = sb[t + o];
      if (ov < sv[t] || (ov == sv[t] && ob < sb[t])) { sv[t] = ov; sb[t] = ob; }
      sa[t] = fmax(sa[t], sa[t + o]);
    }
    __syncthreads();
  }
  const int32_t best = sb[0];
  const double price = sv[0];
  const double absmax = sa[0];
  if (best_out != nullptr && t == 0) *best_out = best;
  if (st == nullptr) return;
  // candidate bookkeeping
  const int32_t r0 = beam_row_ptr[best], r1 = beam_row_ptr[best + 1];
  __shared__ unsigned long long s_hash[256];
  int32_t cnt = 0;
  unsigned long long hsh = 0ull;
  for (int32_t r = r0 + t; r < r1; r += 256) {
    const int32_t l = __ldcg(left + r), rr = __ldcg(right + r);
    cnt += rr - l;
    hsh += leaf_hash(r - r0, l, rr);
  }
  s_cnt[t] = cnt;
  s_hash[t] = hsh;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (t < o) { s_cnt[t] += s_cnt[t + o]; s_hash[t] += s_hash[t + o]; }
    __syncthreads();
  }
  const unsigned long long cand_hash = s_hash[0] + beam_hash(best);
  // duplicate of an aperture already in the pool? (reading S6: counted; it ends the column generation, see below)
  __shared__ int32_t s_dup;
  if (t == 0) s_dup = 0;
  __syncthreads();
  const int32_t K = st->K;
  for (int32_t k = 0; k < K; ++k) {
    if (ap_beam[k] != best || ap_hash[k] != cand_hash) continue;     // hash first (uniform), then verify leaf by leaf
    int32_t diff = 0;
    for (int32_t r = r0 + t; r < r1; r += 256) {
      const int32_t m = r - r0;
      diff |= (ap_left[k * max_rows + m] != __ldcg(left + r)) | (ap_right[k * max_rows + m] != __ldcg(right + r));
    }
    const int any = __syncthreads_or(diff);
    if (!any && t == 0) s_dup = 1;
  }
  __syncthreads();
  if (t == 0) {
    // Optimal iff no aperture has a negative reduced cost.  Numerically (readings S3, S6): the
    // price must be below -price_tol * max|w| * rows.  A candidate identical to a pool aperture k has the reduced
    // cost dF/dy_k of the master, which is >= 0 at the master's optimum: its negative price is residue of the
    // master solve and, being the minimum over all apertures, bounds every other reduced cost.  It proves
    // optimality only if that solve CONVERGED and the residue is of the size the solve reports (10 x its KKT
    // residual, or the price tolerance); otherwise the run is STALLED (done = 2): appending the column again
    // cannot help, and optimality is not claimed.
    const double tol_abs = price_tol * absmax * (double)(r1 - r0);
    const bool improving = price < -tol_abs;
    int done = improving ? 0 : 1;
    if (improving && s_dup) done = (!st->m_hit_max && -price <= 10.0 * fmax(st->m_kkt, tol_abs)) ? 1 : 2;
    if (improving && s_dup) st->n_duplicates += 1;   // as the oracle's driver: the ordinary converged stop is not a duplicate event
    st->cand_beam = best;
    st->cand_hash = cand_hash;
    st->cand_price = price;
    st->w_abs_max = absmax;
    st->cand_nopen = s_cnt[0];
    st->cand_dup = s_dup;
    st->done = done;
    st->cand_valid = (done == 0 && K < k_max) ? 1 : 0;
  }
}

__global__ void __launch_bounds__(256) k_price_select(const double *beam_price, const double *beam_absmax, int32_t n_beams,
                                                      const int32_t *beam_row_ptr, const int32_t *left,
                                                      const int32_t *right, int32_t *best_out, DevState *st,
                                                      double price_tol, int32_t k_max, int32_t max_rows,
                                                      const int32_t *ap_beam, const int32_t *ap_left,
                                                      const int32_t *ap_right, const unsigned long long *ap_hash) {
  price_select_body(beam_price, beam_absmax, n_beams, beam_row_ptr, left, right, best_out, st, price_tol, k_max, max_rows,
                    ap_beam, ap_left, ap_right, ap_hash);
}

// the candidate becomes column K of the pool tables; its 0/1 beamlet mask is the x of step 7 (a_K = D 1_A)
__device__ void append_body(int32_t i0, int32_t stride, const DevState *st, int32_t n_bl, int32_t max_rows,
                            const int32_t *__restrict__ bl_row, const int32_t *__restrict__ row_beam,
                            const int32_t *__restrict__ beam_row_ptr, const int32_t *__restrict__ row_bl_ptr,
                            const int32_t *left, const int32_t *right, int32_t *ap_beam, int32_t *ap_left,
                            int32_t *ap_right, unsigned long long *ap_hash, float *xmask) {
  if (!st->cand_valid) return;
  const int32_t K = st->K, b = st->cand_beam;
  const int32_t r0 = beam_row_ptr[b], nr = beam_row_ptr[b + 1] - r0;
  const int32_t n = (xmask != nullptr && n_bl > max_rows) ? n_bl : max_rows;
  for (int32_t i = i0; i < n; i += stride) {
    if (xmask != nullptr && i < n_bl) {
      const int32_t r = bl_row[i];
      float m = 0.f;
      if (row_beam[r] == b) {
        const int32_t c = i - row_bl_ptr[r];
        m = (c >= __ldcg(left + r) && c < __ldcg(right + r)) ? 1.f : 0.f;
      }
      xmask[i] = m;
    }
    if (i == 0) { ap_beam[K] = b; ap_hash[K] = st->cand_hash; }
    if (i < max_rows) {
      ap_left[K * max_rows + i] = i < nr ? __ldcg(left + r0 + i) : 0;
      ap_right[K * max_rows + i] = i < nr ? __ldcg(right + r0 + i) : 0;
    }
  }
}

__device__ void price_tail(const PriceTail &q) {
  __shared__ bool s_last;
  const int t = threadIdx.x;
  __threadfence();
  __syncthreads();
  if (t == 0) s_last = atomicAdd(q.ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!s_last) return;
  if (t == 0) *q.ticket = 0u;
  __threadfence();
  if (q.do_beams) {
    for (int b = t >> 5; b < q.n_beams; b += 8) price_beam_body(b, q.vstar, q.row_absmax, q.beam_row_ptr, q.beam_price, q.beam_absmax);
    __threadfence_block();
    __syncthreads();
  }
  price_select_body(q.beam_price, q.beam_absmax, q.n_beams, q.beam_row_ptr, q.left, q.right, q.best_out, q.st, q.price_tol,
                    q.k_max, q.max_rows, q.ap_beam, q.ap_left, q.ap_right, q.ap_hash);
  if (q.st == nullptr) return;
  __threadfence_block();
  __syncthreads();
  append_body(t, 256, q.st, q.n_bl, q.max_rows, q.bl_row, q.row_beam, q.beam_row_ptr, q.row_bl_ptr, q.left, q.right, q.ap_beam,
              q.ap_left, q.ap_right, q.ap_hash, q.xmask);
}

size_t chain_pricing_smem(int32_t max_rows, int32_t width) {
  const size_t S = (size_t)(width + 1) * (size_t)(width + 1);
  return align_up((size_t)max_rows * (size_t)(width + 1) * 8 + 3 * S * 8 + S * 4, 16);
}

cudaError_t launch_pricing(Ctx *c, const float *w, const int32_t *row_bl_ptr, const int32_t *beam_row_ptr,
                           int32_t n_rows, int32_t n_beams, int32_t *left, int32_t *right, double *vstar,
                           double *row_absmax, double *beam_price, double *beam_absmax, int32_t *best_out,
                           bool update_state, int32_t max_row_len) {
  const int wpb = 8;
  PriceTail tl{};
  tl.ticket = &c->d.state->ticket_misc;
  tl.n_beams = n_beams; tl.n_rows = n_rows; tl.n_bl = c->n_bl; tl.max_rows = c->max_rows_per_beam; tl.k_max = c->opt.k_max;
  tl.beam_row_ptr = beam_row_ptr; tl.row_bl_ptr = row_bl_ptr; tl.bl_row = c->d.bl_row; tl.row_beam = c->d.row_beam;
  tl.vstar = vstar; tl.row_absmax = row_absmax; tl.beam_price = beam_price; tl.beam_absmax = beam_absmax;
  tl.left = left; tl.right = right; tl.best_out = best_out;
  tl.st = update_state ? c->d.state : nullptr;
  tl.price_tol = c->opt.price_tol;
  tl.ap_beam = c->d.ap_beam; tl.ap_left = c->d.ap_left; tl.ap_right = c->d.ap_right; tl.ap_hash = c->d.ap_hash;
  tl.xmask = spmv_builds_mask(c) ? nullptr : c->d.xmask;
  c->cand_appended = false;
  if (c->opt.mlc_mode == DAO_MLC_JAWS_ONLY) {
    // the context's own MLC tables only (dao_price_from_w refuses caller tables in this mode)
    const size_t smem = (size_t)c->max_rows_per_beam * (size_t)(c->max_beam_width + 1) * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(k_price_jaws, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ++c->n_launches;
    k_price_jaws<<<n_beams, 256, smem, c->stream>>>(w, beam_row_ptr, row_bl_ptr, c->d.row_col0, c->max_beam_width, vstar,
                                                    left, right, beam_price, beam_absmax, tl);
    c->cand_appended = update_state;
    return cudaGetLastError();
  }
  if (c->opt.mlc_mode == DAO_MLC_INTERDIGITATION || c->opt.mlc_mode == DAO_MLC_CONNECTED) {
    const size_t smem = chain_pricing_smem(c->max_rows_per_beam, c->max_beam_width);
    cudaError_t e = cudaFuncSetAttribute(k_price_chain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ++c->n_launches;
    k_price_chain<<<n_beams, 256, smem, c->stream>>>(c->opt.mlc_mode, w, beam_row_ptr, row_bl_ptr, c->d.row_col0,
                                                     c->max_beam_width, c->max_rows_per_beam, c->d.chain_from, vstar, left, right,
                                                     beam_price, beam_absmax, tl);
    c->cand_appended = update_state;
    return cudaGetLastError();
  }
  // max_row_len > 0: known on the host (the context's own tables); < 0: caller tables, decided on the device
  const bool seq_possible = n_rows >= kPriceSeqMinRows && max_row_len != 0;
  if (!seq_possible && n_rows > 0) {
    // the usual case (a few hundred leaf rows): ONE launch, warp per row + the tail in the last CTA
    tl.do_beams = 1;
    ++c->n_launches;
    k_price_rows<<<(n_rows + wpb - 1) / wpb, wpb * 32, 0, c->stream>>>(w, row_bl_ptr, n_rows, vstar, left, right, row_absmax,
                                                                      nullptr, tl);
    c->cand_appended = update_state;
    return cudaGetLastError();
  }
  // many rows (the 10^4-10^5-row end of configs[3]): thread-per-row kernel where the rows are short enough, separate
  // beam-sum and selection launches
  PriceTail none{};
  const int32_t *flag = nullptr;
  if (seq_possible && max_row_len < 0) {
    int32_t *f = &c->d.state->price_maxlen;
    cudaError_t e = cudaMemsetAsync(f, 0, sizeof(int32_t), c->stream);
    if (e != cudaSuccess) return e;
    ++c->n_launches;
    k_price_maxlen<<<std::min((n_rows + 255) / 256, c->n_sm * 4), 256, 0, c->stream>>>(row_bl_ptr, n_rows, f);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    flag = f;
  }
  if (seq_possible && (flag || max_row_len <= kPriceSeqMaxLen)) {
    ++c->n_launches;
    k_price_rows_seq<<<(n_rows + 127) / 128, 128, 0, c->stream>>>(w, row_bl_ptr, n_rows, vstar, left, right, row_absmax, flag);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (n_rows > 0 && (!seq_possible || flag || max_row_len > kPriceSeqMaxLen)) {
    ++c->n_launches;
    k_price_rows<<<(n_rows + wpb - 1) / wpb, wpb * 32, 0, c->stream>>>(w, row_bl_ptr, n_rows, vstar, left, right, row_absmax,
                                                                      flag, none);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  ++c->n_launches;
  k_price_beams<<<(n_beams + wpb - 1) / wpb, wpb * 32, 0, c->stream>>>(vstar, row_absmax, beam_row_ptr, n_beams, beam_price,
                                                                       beam_absmax);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  ++c->n_launches;
  k_price_select<<<1, 256, 0, c->stream>>>(beam_price, beam_absmax, n_beams, beam_row_ptr, left, right, best_out,
                                           update_state ? c->d.state : nullptr, c->opt.price_tol, c->opt.k_max,
                                           c->max_rows_per_beam, c->d.ap_beam, c->d.ap_left, c->d.ap_right, c->d.ap_hash);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Append the pending candidate to the pool tables at index K and write its 0/1 beamlet mask
// (the x of step 7, a_K = D 1_A).  The pool size itself is advanced by the master kernel.
// ------------------------------------------------------------------------------------------
__global__ void k_append_candidate(const DevState *st, int32_t n_bl, int32_t max_rows, const int32_t *bl_row,
                                   const int32_t *row_beam, const int32_t *beam_row_ptr, const int32_t *row_bl_ptr,
                                   const int32_t *left, const int32_t *right, int32_t *ap_beam, int32_t *ap_left,
                                   int32_t *ap_right, unsigned long long *ap_hash, float *xmask) {
  append_body(blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, st, n_bl, max_rows, bl_row, row_beam,
              beam_row_ptr, row_bl_ptr, left, right, ap_beam, ap_left, ap_right, ap_hash, xmask);
}

cudaError_t launch_append_candidate(Ctx *c) {
  if (c->cand_appended) {                 // the pricing launch already appended its winner (price_tail)
    c->cand_appended = false;
    return cudaSuccess;
  }
  const int t = 128;
  const int n = c->n_bl > c->max_rows_per_beam ? c->n_bl : c->max_rows_per_beam;
  ++c->n_launches;
  k_append_candidate<<<(n + t - 1) / t, t, 0, c->stream>>>(c->d.state, c->n_bl, c->max_rows_per_beam, c->d.bl_row,
                                                           c->d.row_beam, c->d.beam_row_ptr, c->d.row_bl_ptr,
                                                           c->d.left, c->d.right, c->d.ap_beam, c->d.ap_left,
                                                           c->d.ap_right, c->d.ap_hash, c->d.xmask);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// dao_price_from_w_static: steps 5-6 for a caller that has no context and may not allocate (a host process whose
// device memory is owned by someone else, or whose rules forbid cudaMalloc / cudaFree at run time -- see dao.h).
// Same row kernel body and same last-CTA tail as the one-launch path of launch_pricing; what that path keeps in the
// context's workspace sits in this fixed array of the library image instead:
//     [0, 256)                        ticket counter of the tail (uint32, the rest of the line unused)
//     [256, 256 + 8 MAX_ROWS)         max |w| per leaf row   (double)
//     [.., .. + 8 MAX_BEAMS)          max |w| per beam       (double)
// One copy per GPU that loads the library, for the life of the process.  In HOST code the name below is only a
// handle for cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel as one; the
// host side looks the address up once per device and passes that pointer.
// ------------------------------------------------------------------------------------------
constexpr size_t kStaticTicketBytes = 256;
constexpr size_t kStaticScratchBytes = DAO_STATIC_SCRATCH_BYTES;
static_assert(kStaticScratchBytes == kStaticTicketBytes + 8 * (size_t)DAO_STATIC_MAX_ROWS + 8 * (size_t)DAO_STATIC_MAX_BEAMS,
              "dao.h and the scratch layout disagree");
static_assert(DAO_STATIC_MAX_ROWS < kPriceSeqMinRows, "the static entry point only has the one-launch kernel");
static __device__ __align__(256) unsigned char g_static_price_scratch[kStaticScratchBytes];

__global__ void __launch_bounds__(256) k_price_rows_static(const float *w, const int32_t *row_bl_ptr,
                                                           const int32_t *beam_row_ptr, int32_t n_rows, int32_t n_beams,
                                                           double *vstar, int32_t *left, int32_t *right,
                                                           double *beam_price, int32_t *best_out, unsigned char *scratch) {
  double *row_absmax = reinterpret_cast<double *>(scratch + kStaticTicketBytes);
  double *beam_absmax = row_absmax + DAO_STATIC_MAX_ROWS;
  price_rows_body(w, row_bl_ptr, n_rows, vstar, left, right, row_absmax, nullptr);
  PriceTail q{};                       // st = null: beam sums and the best beam, no candidate bookkeeping
  q.ticket = reinterpret_cast<uint32_t *>(scratch);
  q.do_beams = 1;
  q.n_beams = n_beams; q.n_rows = n_rows;
  q.beam_row_ptr = beam_row_ptr; q.row_bl_ptr = row_bl_ptr;
  q.vstar = vstar; q.row_absmax = row_absmax; q.beam_price = beam_price; q.beam_absmax = beam_absmax;
  q.left = left; q.right = right; q.best_out = best_out;
  price_tail(q);
}

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mutex;
static unsigned char *g_static_scratch_of_device[kStaticMaxDevices];   // device address of the array, per device

dao_status price_from_w_static(const float *w, const int32_t *row_bl_ptr, const int32_t *beam_row_ptr, int32_t n_rows,
                               int32_t n_beams, int32_t *left, int32_t *right, double *vstar, double *beam_price,
                               int32_t *best_out, cudaStream_t stream, std::string *err) {
  if (!w || !row_bl_ptr || !beam_row_ptr || !left || !right || !vstar || !beam_price || !best_out) {
    *err = "dao_price_from_w_static: null pointer";
    return DAO_E_ARG;
  }
  if (n_rows < 1 || n_beams < 1) {
    *err = "dao_price_from_w_static: n_rows and n_beams must be >= 1";
    return DAO_E_ARG;
  }
  if (n_rows > DAO_STATIC_MAX_ROWS || n_beams > DAO_STATIC_MAX_BEAMS) {
    *err = "dao_price_from_w_static: " + std::to_string(n_rows) + " leaf rows / " + std::to_string(n_beams) +
           " beams exceed the fixed scratch array (DAO_STATIC_MAX_ROWS = " + std::to_string(DAO_STATIC_MAX_ROWS) +
           ", DAO_STATIC_MAX_BEAMS = " + std::to_string(DAO_STATIC_MAX_BEAMS) +
           "); use dao_price_from_w with a context for larger problems";
    return DAO_E_SHAPE;
  }
  auto cuda_fail = [&](const char *what, cudaError_t e) {
    *err = std::string("dao_price_from_w_static: ") + what + ": " + cudaGetErrorString(e);
    return DAO_E_CUDA;
  };
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail("cudaGetDevice", e);
  if (dev < 0 || dev >= kStaticMaxDevices) {
    *err = "dao_price_from_w_static: device ordinal beyond the per-device address table";
    return DAO_E_UNSUPPORTED;
  }
  unsigned char *scratch = nullptr;
  {
    // set-up, once per device, with that device current: the array's address on THIS device
    std::lock_guard<std::mutex> lock(g_static_mutex);
    scratch = g_static_scratch_of_device[dev];
    if (scratch == nullptr) {
      e = cudaGetSymbolAddress(reinterpret_cast<void **>(&scratch), g_static_price_scratch);
      if (e != cudaSuccess) return cuda_fail("cudaGetSymbolAddress", e);
      if (scratch == nullptr) return cuda_fail("cudaGetSymbolAddress returned a null address", cudaErrorInvalidSymbol);
      g_static_scratch_of_device[dev] = scratch;
    }
  }
  // the array keeps the last call's contents: the ticket must start at zero (a launch that died half way would
  // otherwise leave it counting); the two max|w| arrays are written in full before the tail reads them
  e = cudaMemsetAsync(scratch, 0, kStaticTicketBytes, stream);
  if (e != cudaSuccess) return cuda_fail("cudaMemsetAsync", e);
  const int wpb = 8;
  k_price_rows_static<<<(n_rows + wpb - 1) / wpb, wpb * 32, 0, stream>>>(w, row_bl_ptr, beam_row_ptr, n_rows, n_beams, vstar,
                                                                        left, right, beam_price, best_out, scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("k_price_rows_static", e);
  return DAO_OK;
}

}  // namespace dao
