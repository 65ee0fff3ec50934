/*
 * dao_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded fp64 CPU statement of what the column-generation direct aperture
 * optimisation (DAO) hot path of Men, Jia & Jiang (arXiv 1003.5402) computes.  Written from
 * /root/reference/PAPER.md only.  It shares no code, header, table or helper with the CUDA
 * library under paper_1003_5402_b200/csrc/ and must never be linked, imported or executed by the
 * product path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.
 *
 * Conventions:
 *   D is stored voxel-major: row j = voxel, column i = beamlet (the paper writes D_ij with i the
 *   beamlet).  val is fp32 as handed to both implementations; everything else here
 *   is fp64.  Beamlets are numbered beam-major, then leaf row, then left to right.
 *   Leaf positions are reported 0-based half-open [left, right) inside the leaf row:
 *   left = l*, right = r* - 1 in the paper's 1-based notation (open beamlets l*+1 .. r*-1,
 *   PAPER.md:140, 156-165); a closed row is (0, 0) = the paper's initial (l*, r*) = (0, 1).
 *
 * Pins: every function below is pinned by tests/test_oracle_*.py against something other than
 * itself (dense numpy products, closed forms, finite differences, O(n^2)/exhaustive enumeration,
 * scipy.optimize.nnls, bisection, KKT conditions).  No function is "parity unpinned"; the only
 * unpinned item is agreement with the paper's Table 1 numbers, which need clinical data.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ O1: dose, eq. (1) with (2),(7)
 * z_j = sum_i D_ji x_i  (eq. 1 with D_kj = sum_{i in A_k} D_ij, eq. 2, and
 * x_i = sum_{k in K_i} y_k, eq. 7). */
void orc_dose(int32_t n_vox, const int32_t *row_ptr, const int32_t *col_idx, const float *val,
              const double *x, double *z)
{
    for (int32_t j = 0; j < n_vox; ++j) {
        double s = 0.0;
        for (int32_t e = row_ptr[j]; e < row_ptr[j + 1]; ++e)
            s += (double)val[e] * x[col_idx[e]];
        z[j] = s;
    }
}

/* ------------------------------------------------------------------ eq. (7): beamlet intensities
 * x_i = sum over apertures k that contain beamlet i of y_k.
 * Aperture k lives in beam ap_beam[k]; its leaves are ap_left/ap_right[k*max_rows + m] for the
 * m-th leaf row of that beam, half-open column offsets inside the row. */
void orc_beamlet_intensity(int32_t n_bl, int32_t n_ap, const int32_t *ap_beam, const int32_t *ap_left,
                           const int32_t *ap_right, int32_t max_rows, const double *y,
                           const int32_t *beam_row_ptr, const int32_t *row_bl_ptr, double *x)
{
    for (int32_t i = 0; i < n_bl; ++i) x[i] = 0.0;
    for (int32_t k = 0; k < n_ap; ++k) {
        int32_t b = ap_beam[k];
        for (int32_t r = beam_row_ptr[b]; r < beam_row_ptr[b + 1]; ++r) {
            int32_t m = r - beam_row_ptr[b];
            for (int32_t c = ap_left[k * max_rows + m]; c < ap_right[k * max_rows + m]; ++c)
                x[row_bl_ptr[r] + c] += y[k];
        }
    }
}

/* ------------------------------------------------------------------ per-voxel penalty parameters
 * eq. (9)-(10): structure s contributes alpha_s/|v_s| (under, targets only) and
 * beta_s/|v_s| (over) per voxel; |v_s| = number of voxels labelled s.  Voxels labelled -1 carry
 * no penalty.  Output arrays have length n_vox: a_j, b_j, tm_j (= T_s^-), tp_j (= T_s^+). */
void orc_voxel_params(int32_t n_vox, const int32_t *vox_struct, int32_t n_struct,
                      const double *t_under, const double *w_under, const double *t_over,
                      const double *w_over, double *a, double *b, double *tm, double *tp)
{
    double *cnt = (double *)calloc((size_t)(n_struct > 0 ? n_struct : 1), sizeof(double));
    for (int32_t j = 0; j < n_vox; ++j)
        if (vox_struct[j] >= 0) cnt[vox_struct[j]] += 1.0;
    for (int32_t j = 0; j < n_vox; ++j) {
        int32_t s = vox_struct[j];
        if (s < 0) { a[j] = b[j] = 0.0; tm[j] = tp[j] = 0.0; continue; }
        a[j] = w_under[s] / cnt[s];
        b[j] = w_over[s] / cnt[s];
        tm[j] = t_under[s];
        tp[j] = t_over[s];
    }
    free(cnt);
}

/* ------------------------------------------------------------------ O2: objective, eq. (3)-(5), (9)-(10)
 * F(z) = sum_j [ a_j max(0, T_j^- - z_j)^2 + b_j max(0, z_j - T_j^+)^2 ]. */
double orc_objective(int32_t n_vox, const double *z, const double *a, const double *b,
                     const double *tm, const double *tp)
{
    double f = 0.0;
    for (int32_t j = 0; j < n_vox; ++j) {
        double u = tm[j] - z[j]; if (u < 0.0) u = 0.0;
        double o = z[j] - tp[j]; if (o < 0.0) o = 0.0;
        f += a[j] * u * u + b[j] * o * o;
    }
    return f;
}

/* ------------------------------------------------------------------ O3: voxel gradient = dual multiplier pi_j
 * pi_j = dF/dz_j = -2 a_j max(0, T_j^- - z_j) + 2 b_j max(0, z_j - T_j^+)  (reading S1). */
void orc_voxel_gradient(int32_t n_vox, const double *z, const double *a, const double *b,
                        const double *tm, const double *tp, double *g)
{
    for (int32_t j = 0; j < n_vox; ++j) {
        double u = tm[j] - z[j]; if (u < 0.0) u = 0.0;
        double o = z[j] - tp[j]; if (o < 0.0) o = 0.0;
        g[j] = -2.0 * a[j] * u + 2.0 * b[j] * o;
    }
}

/* ------------------------------------------------------------------ O4: beamlet gradient
 * w_i = sum_j D_ij pi_j, computed straight from the voxel-major CSR (no transposed copy). */
void orc_beamlet_gradient(int32_t n_vox, int32_t n_bl, const int32_t *row_ptr, const int32_t *col_idx,
                          const float *val, const double *g, double *w)
{
    for (int32_t i = 0; i < n_bl; ++i) w[i] = 0.0;
    for (int32_t j = 0; j < n_vox; ++j)
        for (int32_t e = row_ptr[j]; e < row_ptr[j + 1]; ++e)
            w[col_idx[e]] += (double)val[e] * g[j];
}

/* ------------------------------------------------------------------ O5: one leaf row, plain definition
 * Over all 0 <= l <= r <= n minimise sum_{i=l+1..r} w_i (1-based beamlets; l = r is the closed row,
 * value 0).  Ties: smallest l, then smallest r; the closed row wins every tie at value 0 and is
 * reported as (0, 0).  O(n^2) double loop; sums accumulated left to right.  (PAPER.md:140.) */
void orc_price_row_exhaustive(int32_t n, const double *w, double *vstar, int32_t *left, int32_t *right)
{
    double best = 0.0; int32_t bl = 0, br = 0;
    for (int32_t l = 0; l < n; ++l) {
        double s = 0.0;
        for (int32_t r = l + 1; r <= n; ++r) {
            s += w[r - 1];
            if (s < best) { best = s; bl = l; br = r; }   /* strict: earlier (l, r) wins ties */
        }
    }
    *vstar = best; *left = bl; *right = br;
}

/* The paper's single left-to-right scan, transcribed literally:
 *   v = vbar = v* = 0; l = l* = 0; r = r* = 1
 *   1. v = v + w_r   2. if v > vbar: vbar = v, l = r   3. if v - vbar < v*: v* = v - vbar, l* = l, r* = r+1
 *   4. if r < n: r = r+1, goto 1; else stop.
 * Returns the ABI convention left = l*, right = r* - 1. */
void orc_price_row_scan(int32_t n, const double *w, double *vstar, int32_t *left, int32_t *right)
{
    double v = 0.0, vbar = 0.0, vs = 0.0;
    int32_t l = 0, ls = 0, r = 1, rs = 1;
    while (n > 0) {
        v = v + w[r - 1];
        if (v > vbar) { vbar = v; l = r; }
        if (v - vbar < vs) { vs = v - vbar; ls = l; rs = r + 1; }
        if (r < n) r = r + 1; else break;
    }
    *vstar = vs; *left = ls; *right = rs - 1;
}

/* ------------------------------------------------------------------ O5+O6: pricing sub-problem, eq. (8)
 * Every leaf row by its plain definition, price_b = sum of the row minima of beam b
 * (PAPER.md:169), best beam = smallest price, ties to the smallest beam index (reading S4). */
void orc_price(const double *w, int32_t n_beams, const int32_t *beam_row_ptr, const int32_t *row_bl_ptr,
               double *vstar, int32_t *left, int32_t *right, double *beam_price, int32_t *best_beam)
{
    int32_t bb = -1;
    for (int32_t b = 0; b < n_beams; ++b) {
        double p = 0.0;
        for (int32_t r = beam_row_ptr[b]; r < beam_row_ptr[b + 1]; ++r) {
            orc_price_row_exhaustive(row_bl_ptr[r + 1] - row_bl_ptr[r], w + row_bl_ptr[r],
                                     &vstar[r], &left[r], &right[r]);
            p += vstar[r];
        }
        beam_price[b] = p;
        if (bb < 0 || p < beam_price[bb]) bb = b;
    }
    *best_beam = bb;
}

/* ------------------------------------------------------------------ O7: aperture dose column, eq. (2)
 * a_j = sum_{i in A} D_ij  with `open[i]` = 1 for the beamlets of the aperture. */
void orc_aperture_column(int32_t n_vox, const int32_t *row_ptr, const int32_t *col_idx, const float *val,
                         const uint8_t *open, double *a)
{
    for (int32_t j = 0; j < n_vox; ++j) {
        double s = 0.0;
        for (int32_t e = row_ptr[j]; e < row_ptr[j + 1]; ++e)
            if (open[col_idx[e]]) s += (double)val[e];
        a[j] = s;
    }
}

/* ------------------------------------------------------------------ O8: restricted master problem
 * min_{y >= 0} F(A y),  A = [a_0 .. a_{K-1}] (aperture-major: A[k*n_vox + j]).
 *
 * The paper names the method (gradient projection, Bazaraa et al.) but gives no step rule, stopping
 * rule or tolerance (reading S2).  The RESULT has a plain definition: F is convex, so any y >= 0
 * meeting the KKT conditions (grad_k >= 0, grad_k = 0 where y_k > 0) attains the unique optimal
 * value.  Two plain methods are provided; the tests check both against KKT, bisection (K = 1),
 * scipy NNLS (least-squares special case) and each other.
 *
 * Shared pieces ------------------------------------------------------------------------------- */
static void master_dose(int32_t n_vox, int32_t K, const double *A, const double *y, double *z)
{
    for (int32_t j = 0; j < n_vox; ++j) z[j] = 0.0;
    for (int32_t k = 0; k < K; ++k) {
        const double *ak = A + (size_t)k * n_vox;
        if (y[k] != 0.0)
            for (int32_t j = 0; j < n_vox; ++j) z[j] += y[k] * ak[j];
    }
}

static double dphi(int32_t n_vox, const double *z, const double *dz, double t, const double *a,
                   const double *b, const double *tm, const double *tp)
{   /* d/dt F(z + t dz) */
    double s = 0.0;
    for (int32_t j = 0; j < n_vox; ++j) {
        if (dz[j] == 0.0) continue;
        double zz = z[j] + t * dz[j];
        double u = tm[j] - zz; if (u < 0.0) u = 0.0;
        double o = zz - tp[j]; if (o < 0.0) o = 0.0;
        s += dz[j] * (-2.0 * a[j] * u + 2.0 * b[j] * o);
    }
    return s;
}

/* Exact minimiser of the convex piecewise-quadratic t -> F(z + t dz) on [0, t_max] given
 * dphi(0) < 0: t_max if the slope is still <= 0 there, else the root of the non-decreasing
 * piecewise-linear slope by bisection to full fp64 resolution. */
static double exact_step(int32_t n_vox, const double *z, const double *dz, double t_max,
                         const double *a, const double *b, const double *tm, const double *tp,
                         int *hit_bound)
{
    double lo = 0.0, hi;
    *hit_bound = 0;
    if (isfinite(t_max)) {
        if (dphi(n_vox, z, dz, t_max, a, b, tm, tp) <= 0.0) { *hit_bound = 1; return t_max; }
        hi = t_max;
    } else {
        hi = 1.0;
        int guard = 0;
        while (dphi(n_vox, z, dz, hi, a, b, tm, tp) < 0.0 && guard++ < 200) hi *= 2.0;
    }
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;
        if (dphi(n_vox, z, dz, mid, a, b, tm, tp) < 0.0) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

static double kkt_residual(int32_t K, const double *y, const double *grad)
{   /* max over k of |grad_k| where y_k > 0, and of max(0, -grad_k) where y_k = 0 */
    double r = 0.0;
    for (int32_t k = 0; k < K; ++k) {
        double v = (y[k] > 0.0) ? fabs(grad[k]) : (grad[k] < 0.0 ? -grad[k] : 0.0);
        if (v > r) r = v;
    }
    return r;
}

static double ymax1(int32_t K, const double *y)
{
    double m = 1.0;
    for (int32_t k = 0; k < K; ++k) if (y[k] > m) m = y[k];
    return m;
}

/* Method 1: gradient projection (Rosen / Bazaraa et al., the method the paper names)
 * with exact line search.  Direction p_k = -grad_k, except p_k = 0 where y_k = 0 and grad_k > 0
 * (the projection of the steepest-descent direction onto the feasible cone); step = exact
 * minimiser along the feasible ray, capped at the first bound.  Stops when
 *   max_k |p_k| * max(1, max y) <= tol * max(F, 1e-300)     or after max_iter iterations.
 * Returns the number of iterations; *f_out = F(A y), *kkt_out = KKT residual at return. */
int32_t orc_master_pg(int32_t n_vox, int32_t K, const double *A, double *y, const double *a,
                      const double *b, const double *tm, const double *tp, double tol,
                      int32_t max_iter, double *f_out, double *kkt_out)
{
    double *z = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *g = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *dz = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *grad = (double *)malloc(sizeof(double) * (size_t)(K > 0 ? K : 1));
    double *p = (double *)malloc(sizeof(double) * (size_t)(K > 0 ? K : 1));
    int32_t it = 0;
    double f = 0.0;
    for (;;) {
        master_dose(n_vox, K, A, y, z);
        f = orc_objective(n_vox, z, a, b, tm, tp);
        orc_voxel_gradient(n_vox, z, a, b, tm, tp, g);
        double pmax = 0.0;
        for (int32_t k = 0; k < K; ++k) {
            const double *ak = A + (size_t)k * n_vox;
            double s = 0.0;
            for (int32_t j = 0; j < n_vox; ++j) s += ak[j] * g[j];
            grad[k] = s;
            p[k] = (y[k] <= 0.0 && s > 0.0) ? 0.0 : -s;
            if (fabs(p[k]) > pmax) pmax = fabs(p[k]);
        }
        if (pmax * ymax1(K, y) <= tol * (f > 1e-300 ? f : 1e-300) || it >= max_iter) break;
        double t_max = INFINITY; int32_t kb = -1;
        for (int32_t k = 0; k < K; ++k)
            if (p[k] < 0.0) { double t = y[k] / (-p[k]); if (t < t_max) { t_max = t; kb = k; } }
        master_dose(n_vox, K, A, p, dz);
        int hit = 0;
        double t = exact_step(n_vox, z, dz, t_max, a, b, tm, tp, &hit);
        for (int32_t k = 0; k < K; ++k) { y[k] += t * p[k]; if (y[k] < 0.0) y[k] = 0.0; }
        if (hit && kb >= 0) y[kb] = 0.0;
        ++it;
    }
    *f_out = f; *kkt_out = kkt_residual(K, y, grad);
    free(z); free(g); free(dz); free(grad); free(p);
    return it;
}

/* Method 2: projected Newton on the free variables (semi-smooth Newton for a piecewise-quadratic
 * F) with the same exact line search.  Free set = { k : y_k > 0 or grad_k < 0 }.  On it solve
 * (H + ridge I) d = -grad, H = 2 A_f^T diag(c) A_f with c_j = a_j [z_j < T_j^-] + b_j [z_j > T_j^+]
 * (Gaussian elimination with partial pivoting); fall back to steepest descent when d is not a
 * descent direction.  Same stopping rule as method 1.  Much faster than method 1 on correlated
 * aperture columns; same optimum (convexity), which tests/test_oracle_master.py checks. */
static int solve_dense(int n, double *M, double *rhs)
{   /* in-place Gaussian elimination with partial pivoting; returns 0 on success */
    for (int c = 0; c < n; ++c) {
        int piv = c; double best = fabs(M[c * n + c]);
        for (int r = c + 1; r < n; ++r) if (fabs(M[r * n + c]) > best) { best = fabs(M[r * n + c]); piv = r; }
        if (best == 0.0) return 1;
        if (piv != c) {
            for (int q = 0; q < n; ++q) { double t = M[c * n + q]; M[c * n + q] = M[piv * n + q]; M[piv * n + q] = t; }
            double t = rhs[c]; rhs[c] = rhs[piv]; rhs[piv] = t;
        }
        for (int r = c + 1; r < n; ++r) {
            double f = M[r * n + c] / M[c * n + c];
            if (f == 0.0) continue;
            for (int q = c; q < n; ++q) M[r * n + q] -= f * M[c * n + q];
            rhs[r] -= f * rhs[c];
        }
    }
    for (int c = n - 1; c >= 0; --c) {
        double s = rhs[c];
        for (int q = c + 1; q < n; ++q) s -= M[c * n + q] * rhs[q];
        rhs[c] = s / M[c * n + c];
    }
    return 0;
}

int32_t orc_master_newton(int32_t n_vox, int32_t K, const double *A, double *y, const double *a,
                          const double *b, const double *tm, const double *tp, double tol,
                          int32_t max_iter, double *f_out, double *kkt_out)
{
    double *z = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *g = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *c = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *dz = (double *)malloc(sizeof(double) * (size_t)n_vox);
    size_t Kn = (size_t)(K > 0 ? K : 1);
    double *grad = (double *)malloc(sizeof(double) * Kn);
    double *p = (double *)malloc(sizeof(double) * Kn);
    double *H = (double *)malloc(sizeof(double) * Kn * Kn);
    double *rhs = (double *)malloc(sizeof(double) * Kn);
    int32_t *fr = (int32_t *)malloc(sizeof(int32_t) * Kn);
    int32_t it = 0;
    double f = 0.0;
    for (;;) {
        master_dose(n_vox, K, A, y, z);
        f = orc_objective(n_vox, z, a, b, tm, tp);
        orc_voxel_gradient(n_vox, z, a, b, tm, tp, g);
        double pmax = 0.0; int nf = 0;
        for (int32_t k = 0; k < K; ++k) {
            const double *ak = A + (size_t)k * n_vox;
            double s = 0.0;
            for (int32_t j = 0; j < n_vox; ++j) s += ak[j] * g[j];
            grad[k] = s;
            double pk = (y[k] <= 0.0 && s > 0.0) ? 0.0 : -s;
            if (!(y[k] <= 0.0 && s >= 0.0)) fr[nf++] = k;
            p[k] = pk;
            if (fabs(pk) > pmax) pmax = fabs(pk);
        }
        if (pmax * ymax1(K, y) <= tol * (f > 1e-300 ? f : 1e-300) || it >= max_iter) break;
        /* Newton direction on the free set */
        for (int32_t j = 0; j < n_vox; ++j)
            c[j] = (z[j] < tm[j] ? a[j] : 0.0) + (z[j] > tp[j] ? b[j] : 0.0);
        /* A free variable sitting at 0 whose Newton component is negative cannot move: take it
         * out of the free set and solve again, until the direction is feasible at every bound. */
        int bad = 0, shrunk = 1;
        while (shrunk && nf > 0) {
            double tr = 0.0;
            for (int q = 0; q < nf; ++q)
                for (int r = q; r < nf; ++r) {
                    const double *aq = A + (size_t)fr[q] * n_vox, *ar = A + (size_t)fr[r] * n_vox;
                    double s = 0.0;
                    for (int32_t j = 0; j < n_vox; ++j) s += c[j] * aq[j] * ar[j];
                    H[q * nf + r] = H[r * nf + q] = 2.0 * s;
                    if (q == r) tr += 2.0 * s;
                }
            double ridge = 1e-12 * (tr / nf) + 1e-300;
            for (int q = 0; q < nf; ++q) { H[q * nf + q] += ridge; rhs[q] = -grad[fr[q]]; }
            bad = solve_dense(nf, H, rhs);
            if (bad) break;
            shrunk = 0;
            int m = 0;
            for (int q = 0; q < nf; ++q) {
                if (y[fr[q]] <= 0.0 && rhs[q] < 0.0) { shrunk = 1; continue; }
                fr[m] = fr[q]; rhs[m] = rhs[q]; ++m;
            }
            nf = m;
        }
        double slope = 0.0;
        if (!bad) for (int q = 0; q < nf; ++q) slope += rhs[q] * grad[fr[q]];
        if (!bad && nf > 0 && isfinite(slope) && slope < 0.0) {
            for (int32_t k = 0; k < K; ++k) p[k] = 0.0;
            for (int q = 0; q < nf; ++q) p[fr[q]] = rhs[q];
        }   /* else keep the projected steepest-descent direction p */
        double t_max = INFINITY; int32_t kb = -1;
        for (int32_t k = 0; k < K; ++k)
            if (p[k] < 0.0) { double t = y[k] / (-p[k]); if (t < t_max) { t_max = t; kb = k; } }
        master_dose(n_vox, K, A, p, dz);
        int hit = 0;
        double t = exact_step(n_vox, z, dz, t_max, a, b, tm, tp, &hit);
        for (int32_t k = 0; k < K; ++k) { y[k] += t * p[k]; if (y[k] < 0.0) y[k] = 0.0; }
        if (hit && kb >= 0) y[kb] = 0.0;
        ++it;
    }
    *f_out = f; *kkt_out = kkt_residual(K, y, grad);
    free(z); free(g); free(c); free(dz); free(grad); free(p); free(H); free(rhs); free(fr);
    return it;
}

/* Gradient of the master objective with respect to y at a given y (for KKT checks by the tests
 * and for judging a plan produced elsewhere): grad_k = a_k . pi(A y); returns F(A y). */
double orc_master_gradient(int32_t n_vox, int32_t K, const double *A, const double *y, const double *a,
                           const double *b, const double *tm, const double *tp, double *grad)
{
    double *z = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *g = (double *)malloc(sizeof(double) * (size_t)n_vox);
    master_dose(n_vox, K, A, y, z);
    double f = orc_objective(n_vox, z, a, b, tm, tp);
    orc_voxel_gradient(n_vox, z, a, b, tm, tp, g);
    for (int32_t k = 0; k < K; ++k) {
        const double *ak = A + (size_t)k * n_vox;
        double s = 0.0;
        for (int32_t j = 0; j < n_vox; ++j) s += ak[j] * g[j];
        grad[k] = s;
    }
    free(z); free(g);
    return f;
}

/* ------------------------------------------------------------------ FMO
 * Fluence-map optimisation: the same objective with the beamlet intensities themselves as the
 * decision variables, min_{x >= 0} F(D x) -- "Mathematically, the DAO model is the same as the FMO
 * model ... in which the decision variables are the intensities of all beamlets", solved
 * with "the same gradient projection method".  By eq. (7) every
 * aperture plan is a beamlet plan, so F*_FMO is a lower bound of every DAO objective.
 *
 * Plain gradient projection on the sparse D, the statement of orc_master_pg with A = D^T: direction
 * p_i = -w_i (w = D^T pi, eq. 8's inner sum) except p_i = 0 where x_i = 0 and w_i > 0; exact step along
 * the feasible ray, capped at the first bound.  Stops when max_i |p_i| * max(1, max x) <= tol * F or
 * after max_iter iterations.  Returns the iteration count; *f_out = F(D x), *kkt_out = KKT residual. */
int32_t orc_fmo_pg(int32_t n_vox, int32_t n_bl, const int32_t *row_ptr, const int32_t *col_idx,
                   const float *val, double *x, const double *a, const double *b, const double *tm,
                   const double *tp, double tol, int32_t max_iter, double *f_out, double *kkt_out)
{
    double *z = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *g = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *dz = (double *)malloc(sizeof(double) * (size_t)n_vox);
    double *w = (double *)malloc(sizeof(double) * (size_t)(n_bl > 0 ? n_bl : 1));
    double *p = (double *)malloc(sizeof(double) * (size_t)(n_bl > 0 ? n_bl : 1));
    int32_t it = 0;
    double f = 0.0;
    for (;;) {
        orc_dose(n_vox, row_ptr, col_idx, val, x, z);
        f = orc_objective(n_vox, z, a, b, tm, tp);
        orc_voxel_gradient(n_vox, z, a, b, tm, tp, g);
        orc_beamlet_gradient(n_vox, n_bl, row_ptr, col_idx, val, g, w);
        double pmax = 0.0;
        for (int32_t i = 0; i < n_bl; ++i) {
            p[i] = (x[i] <= 0.0 && w[i] > 0.0) ? 0.0 : -w[i];
            if (fabs(p[i]) > pmax) pmax = fabs(p[i]);
        }
        if (pmax * ymax1(n_bl, x) <= tol * (f > 1e-300 ? f : 1e-300) || it >= max_iter) break;
        double t_max = INFINITY; int32_t ib = -1;
        for (int32_t i = 0; i < n_bl; ++i)
            if (p[i] < 0.0) { double t = x[i] / (-p[i]); if (t < t_max) { t_max = t; ib = i; } }
        orc_dose(n_vox, row_ptr, col_idx, val, p, dz);
        int hit = 0;
        double t = exact_step(n_vox, z, dz, t_max, a, b, tm, tp, &hit);
        for (int32_t i = 0; i < n_bl; ++i) { x[i] += t * p[i]; if (x[i] < 0.0) x[i] = 0.0; }
        if (hit && ib >= 0) x[ib] = 0.0;
        ++it;
    }
    *f_out = f; *kkt_out = kkt_residual(n_bl, x, w);
    free(z); free(g); free(dz); free(w); free(p);
    return it;
}

/* ------------------------------------------------------------------ jaws-only pricing
 * "we are able to handle various MLC hardware constraints ... including standard consecutiveness,
 * interdigitation, connectedness and jaws-only delivery": the paper names the constraint and
 * prints no algorithm.  Reading J1: with jaws only, an aperture of beam b is a RECTANGLE --
 * consecutive leaf rows m1..m2 all opened over the same lateral range [c1, c2), measured in beamlet widths from
 * the beam's leftmost beamlet (row r starts at row_col0[r]), every other row closed; a cell of the rectangle
 * where a row has no beamlet contributes nothing.  The sub-problem (8) becomes: over all rectangles of all
 * beams, minimise the sum of w over the rectangle's beamlets.  Plain definition written out: every rectangle
 * is enumerated in the order c1, c2, m1, m2 (ascending) and replaces the incumbent only when strictly smaller,
 * so the closed aperture (value 0) wins ties at 0 and equal negative values keep the first in that order.
 * Outputs as orc_price: per row the half-open leaves inside the row (closed = (0,0)) and vstar[r] = sum of w
 * over the row's open beamlets; beam_price[b] = value of the best rectangle of beam b. */
void orc_price_jaws(const double *w, int32_t n_beams, const int32_t *beam_row_ptr, const int32_t *row_bl_ptr,
                    const int32_t *row_col0, double *vstar, int32_t *left, int32_t *right, double *beam_price,
                    int32_t *best_beam)
{
    int32_t bb = -1; double bbv = 0.0;
    for (int32_t b = 0; b < n_beams; ++b) {
        const int32_t r0 = beam_row_ptr[b], r1 = beam_row_ptr[b + 1], R = r1 - r0;
        int32_t C = 0;
        for (int32_t r = r0; r < r1; ++r) {
            const int32_t c0 = row_col0 ? row_col0[r] : 0, e = c0 + (row_bl_ptr[r + 1] - row_bl_ptr[r]);
            if (e > C) C = e;
        }
        double best = 0.0; int32_t bc1 = 0, bc2 = 0, bm1 = 0, bm2 = -1;          /* closed */
        double *S = (double *)malloc(sizeof(double) * (size_t)(R > 0 ? R : 1));
        for (int32_t c1 = 0; c1 < C; ++c1)
            for (int32_t c2 = c1 + 1; c2 <= C; ++c2) {
                for (int32_t m = 0; m < R; ++m) {                                /* row sums over [c1, c2) */
                    const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, n = row_bl_ptr[r + 1] - row_bl_ptr[r];
                    const int32_t lo = c1 > c0 ? c1 : c0, hi = c2 < c0 + n ? c2 : c0 + n;
                    double s = 0.0;
                    for (int32_t c = lo; c < hi; ++c) s += w[row_bl_ptr[r] + (c - c0)];
                    S[m] = s;
                }
                for (int32_t m1 = 0; m1 < R; ++m1) {
                    double s = 0.0;
                    for (int32_t m2 = m1; m2 < R; ++m2) {
                        s += S[m2];
                        if (s < best) { best = s; bc1 = c1; bc2 = c2; bm1 = m1; bm2 = m2; }
                    }
                }
            }
        free(S);
        beam_price[b] = best;
        for (int32_t m = 0; m < R; ++m) {
            const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, n = row_bl_ptr[r + 1] - row_bl_ptr[r];
            int32_t lo = bc1 > c0 ? bc1 : c0, hi = bc2 < c0 + n ? bc2 : c0 + n;
            double s = 0.0;
            if (m < bm1 || m > bm2 || hi <= lo) { lo = c0; hi = c0; }
            for (int32_t c = lo; c < hi; ++c) s += w[row_bl_ptr[r] + (c - c0)];
            left[r] = hi > lo ? lo - c0 : 0; right[r] = hi > lo ? hi - c0 : 0; vstar[r] = s;
        }
        if (bb < 0 || best < bbv) { bb = b; bbv = best; }
    }
    *best_beam = bb;
}

/* ------------------------------------------------------------------ interdigitation / connectedness pricing
 * The other two MLC constraints PAPER.md:260 names without an algorithm.  Leaf positions are lateral
 * positions in beamlet widths (row r's beamlets occupy [c0_r, c0_r + n_r)); the state of a row is (a, b),
 * 0 <= a <= b <= W: left leaf tip at a, right leaf tip at b, open cells [a, b), closed when a == b.  An open
 * row stays inside its own beamlets (c0_r <= a < b <= c0_r + n_r); a closed leaf pair may park anywhere.
 *   Reading J2 (mode 2, interdigitation forbidden): for physically adjacent rows m, m+1 a leaf may not pass
 *   the opposing leaf of the neighbouring row:  a_m <= b_{m+1}  and  a_{m+1} <= b_m.
 *   Reading J3 (mode 3, connectedness): the open rows are consecutive and the open intervals of adjacent open
 *   rows share at least one lateral position: max(a_m, a_{m+1}) < min(b_m, b_{m+1}); closed rows are free.
 * The sub-problem minimises the sum of w over the open beamlets of a beam.  The feasible sets are chains over
 * the rows, so the minimum is a shortest path through the layered graph rows x states (the construction of
 * Romeijn et al. 2005 that the paper cites); it is written out as the plain dynamic programme
 *   f_m(s) = val_m(s) + min { f_{m-1}(s') : s' compatible with s },  O(rows x states^2),
 * and pinned against exhaustive enumeration of every aperture on tiny beams.  Several apertures can attain
 * the minimum (closed rows park anywhere; exact ties), so only the VALUE is unique; the aperture returned is
 * the first minimiser in state order and callers compare values and check feasibility. */
static int mlc_compatible(int mode, int a0, int b0, int a1, int b1)
{   /* states of two adjacent rows */
    if (mode == 2) return a0 <= b1 && a1 <= b0;
    /* mode 3: both open -> overlap; otherwise handled by the phase logic of the caller */
    return (a0 > a1 ? a0 : a1) < (b0 < b1 ? b0 : b1);
}

void orc_price_chain(int32_t mode, const double *w, int32_t n_beams, const int32_t *beam_row_ptr,
                     const int32_t *row_bl_ptr, const int32_t *row_col0, double *vstar, int32_t *left,
                     int32_t *right, double *beam_price, int32_t *best_beam)
{
    int32_t bb = -1; double bbv = 0.0;
    for (int32_t bm = 0; bm < n_beams; ++bm) {
        const int32_t r0 = beam_row_ptr[bm], R = beam_row_ptr[bm + 1] - r0;
        int32_t W = 0;
        for (int32_t r = r0; r < r0 + R; ++r) {
            const int32_t e = (row_col0 ? row_col0[r] : 0) + (row_bl_ptr[r + 1] - row_bl_ptr[r]);
            if (e > W) W = e;
        }
        const int32_t S = (W + 1) * (W + 2) / 2;                 /* states (a, b), a <= b, in the order a, then b */
        int32_t *sa = (int32_t *)malloc(sizeof(int32_t) * (size_t)S), *sb = (int32_t *)malloc(sizeof(int32_t) * (size_t)S);
        { int32_t k = 0; for (int32_t a = 0; a <= W; ++a) for (int32_t b = a; b <= W; ++b) { sa[k] = a; sb[k] = b; ++k; } }
        double *f = (double *)malloc(sizeof(double) * (size_t)S * (size_t)(R > 0 ? R : 1));
        int32_t *from = (int32_t *)malloc(sizeof(int32_t) * (size_t)S * (size_t)(R > 0 ? R : 1));
        double best = 0.0; int32_t best_m = -1, best_s = -1;     /* connectedness: best end of an open run */
        for (int32_t m = 0; m < R; ++m) {
            const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0, n = row_bl_ptr[r + 1] - row_bl_ptr[r];
            for (int32_t s = 0; s < S; ++s) {
                const int32_t a = sa[s], b = sb[s];
                double val = 0.0, prev = 0.0; int32_t arg = -1;
                f[(size_t)m * S + s] = INFINITY; from[(size_t)m * S + s] = -1;
                if (a < b) {                                      /* open: inside the row's own beamlets */
                    if (a < c0 || b > c0 + n) continue;
                    for (int32_t c = a; c < b; ++c) val += w[row_bl_ptr[r] + (c - c0)];
                } else if (mode == 3) continue;                   /* connectedness tracks open states only */
                if (m > 0) {
                    prev = (mode == 3) ? 0.0 : INFINITY;          /* mode 3: the run may start at this row */
                    for (int32_t q = 0; q < S; ++q) {
                        const double fq = f[(size_t)(m - 1) * S + q];
                        if (fq == INFINITY || !mlc_compatible(mode, sa[q], sb[q], a, b)) continue;
                        if (fq < prev) { prev = fq; arg = q; }
                    }
                    if (prev == INFINITY) continue;
                }
                f[(size_t)m * S + s] = val + prev; from[(size_t)m * S + s] = arg;
                if (mode == 3 && val + prev < best) { best = val + prev; best_m = m; best_s = s; }
            }
        }
        if (mode == 2) {                                          /* best state of the last row */
            best = INFINITY; best_m = R - 1;
            for (int32_t s = 0; s < S; ++s) if (f[(size_t)(R - 1) * S + s] < best) { best = f[(size_t)(R - 1) * S + s]; best_s = s; }
        }
        for (int32_t r = r0; r < r0 + R; ++r) { left[r] = 0; right[r] = 0; vstar[r] = 0.0; }
        for (int32_t m = best_m, s = best_s; m >= 0 && s >= 0; s = from[(size_t)m * S + s], --m) {
            const int32_t r = r0 + m, c0 = row_col0 ? row_col0[r] : 0;
            if (sa[s] < sb[s]) {
                double val = 0.0;
                for (int32_t c = sa[s]; c < sb[s]; ++c) val += w[row_bl_ptr[r] + (c - c0)];
                left[r] = sa[s] - c0; right[r] = sb[s] - c0; vstar[r] = val;
            }
        }
        beam_price[bm] = best;
        free(sa); free(sb); free(f); free(from);
        if (bb < 0 || best < bbv) { bb = bm; bbv = best; }
    }
    *best_beam = bb;
}
