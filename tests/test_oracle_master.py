"""Pins for the oracle's restricted master problem (O8) and the whole method (O9).

The master's result has a plain definition (the minimum of a convex function over y >= 0), so the
pins are: KKT conditions at return, a 1-D bisection for K = 1, scipy's NNLS on the exact
least-squares special case, scipy L-BFGS-B on the general case, agreement of the two oracle
methods, monotone decrease along column generation, exactness at termination against the master
solved over ALL enumerated apertures, and the FMO lower bound.
"""
import itertools

import numpy as np
import pytest
from scipy.optimize import minimize, nnls

from oracle import dao_oracle as orc


def _params(case):
    return orc.voxel_params(case.vox_struct, case.t_under, case.w_under, case.t_over, case.w_over)


def _random_pool(case, K, seed):
    """K random non-empty apertures -> A [K, n_vox] from the dense matrix."""
    rng = np.random.default_rng(seed)
    A = np.zeros((K, case.n_vox))
    for k in range(K):
        b = int(rng.integers(0, case.n_beams))
        m = np.zeros(case.n_bl)
        for r in range(case.beam_row_ptr[b], case.beam_row_ptr[b + 1]):
            n = case.row_bl_ptr[r + 1] - case.row_bl_ptr[r]
            l = int(rng.integers(0, n)); rr = int(rng.integers(l + 1, n + 1))
            m[case.row_bl_ptr[r] + l: case.row_bl_ptr[r] + rr] = 1.0
        A[k] = case.dense @ m
    return A


def _F_numpy(A, y, vp):
    z = y @ A
    return float(np.sum(vp.a * np.maximum(0, vp.tm - z) ** 2 + vp.b * np.maximum(0, z - vp.tp) ** 2))


def _gradF_numpy(A, y, vp):
    z = y @ A
    g = -2 * vp.a * np.maximum(0, vp.tm - z) + 2 * vp.b * np.maximum(0, z - vp.tp)
    return A @ g


def _assert_kkt(A, res, vp, eps):
    grad = _gradF_numpy(A, res.y, vp)
    scale = max(1.0, float(np.max(np.abs(_gradF_numpy(A, np.zeros_like(res.y), vp)))))
    assert np.all(res.y >= 0.0)
    assert np.all(grad >= -eps * scale), grad.min()
    assert np.all(np.abs(grad[res.y > 0]) <= eps * scale)


@pytest.mark.parametrize("method", ["newton", "pg"])
@pytest.mark.parametrize("K,seed", [(1, 0), (3, 1), (6, 2), (10, 3)])
def test_master_satisfies_kkt_and_matches_lbfgsb(tiny, method, K, seed):
    vp = _params(tiny)
    A = _random_pool(tiny, K, seed)
    res = orc.master(A, np.zeros(K), vp, tol=1e-11, max_iter=200000, method=method)
    _assert_kkt(A, res, vp, 1e-7)
    assert res.objective == pytest.approx(_F_numpy(A, res.y, vp), rel=1e-12)
    ref = minimize(lambda y: _F_numpy(A, y, vp), np.full(K, 0.1), jac=lambda y: _gradF_numpy(A, y, vp),
                   bounds=[(0, None)] * K, method="L-BFGS-B", options={"ftol": 1e-15, "gtol": 1e-12, "maxiter": 5000})
    assert res.objective <= ref.fun * (1 + 1e-9) + 1e-14
    assert res.objective == pytest.approx(ref.fun, rel=1e-6)


def test_master_single_aperture_is_root_of_monotone_slope(tiny):
    """K = 1: phi(y) = F(y a) is a 1-D convex piecewise quadratic; its minimiser is the root of phi'."""
    vp = _params(tiny)
    A = _random_pool(tiny, 1, 11)
    dphi = lambda t: float(_gradF_numpy(A, np.array([t]), vp)[0])
    lo, hi = 0.0, 1.0
    while dphi(hi) < 0:
        hi *= 2
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if dphi(mid) < 0 else (lo, mid)
    for method in ("newton", "pg"):
        res = orc.master(A, np.zeros(1), vp, tol=1e-13, method=method)
        assert res.y[0] == pytest.approx(0.5 * (lo + hi), rel=1e-9)


@pytest.mark.parametrize("method", ["newton", "pg"])
def test_master_least_squares_special_case_equals_nnls(tiny, method):
    """T+ = T-, beta = alpha on targets and T+ = 0 on OARs: F = sum_j c_j (z_j - T_j)^2 exactly
    (z >= 0 always), so the optimum equals scipy.optimize.nnls on (sqrt(c) A^T, sqrt(c) T)."""
    t_under = np.array([1.0, 0.0]); w_under = np.array([10.0, 0.0])
    t_over = np.array([1.0, 0.0]); w_over = np.array([10.0, 2.0])
    vp = orc.voxel_params(tiny.vox_struct, t_under, w_under, t_over, w_over)
    K = 8
    A = _random_pool(tiny, K, 5)
    c = vp.b.copy()                       # a = b on targets, a = 0 / b > 0 on OARs, 0 elsewhere
    T = vp.tp.copy()
    M = (np.sqrt(c)[:, None] * A.T)
    y_ref, rnorm = nnls(M, np.sqrt(c) * T, maxiter=10000)
    res = orc.master(A, np.zeros(K), vp, tol=1e-12, max_iter=500000, method=method)
    assert res.objective == pytest.approx(rnorm ** 2, rel=1e-8)
    assert _F_numpy(A, y_ref, vp) == pytest.approx(rnorm ** 2, rel=1e-10)


def test_master_methods_agree_from_warm_start(tiny):
    vp = _params(tiny)
    A = _random_pool(tiny, 7, 21)
    rng = np.random.default_rng(0)
    y0 = rng.random(7) * 0.2
    a = orc.master(A, y0, vp, tol=1e-12, max_iter=500000, method="pg")
    b = orc.master(A, y0, vp, tol=1e-12, method="newton")
    assert a.objective == pytest.approx(b.objective, rel=1e-9)
    f, grad = orc.master_gradient(A, b.y, vp)
    assert f == pytest.approx(b.objective, rel=1e-13)
    np.testing.assert_allclose(grad, _gradF_numpy(A, b.y, vp), rtol=1e-10, atol=1e-13)


# ----------------------------------------------------------------------------- O9
def _all_apertures(case):
    cols, meta = [], []
    for b in range(case.n_beams):
        rows = range(case.beam_row_ptr[b], case.beam_row_ptr[b + 1])
        per_row = []
        for r in rows:
            n = case.row_bl_ptr[r + 1] - case.row_bl_ptr[r]
            per_row.append([(0, 0)] + [(l, rr) for l in range(n) for rr in range(l + 1, n + 1)])
        for combo in itertools.product(*per_row):
            if all(c == (0, 0) for c in combo):
                continue
            m = np.zeros(case.n_bl)
            for r, (l, rr) in zip(rows, combo):
                m[case.row_bl_ptr[r] + l: case.row_bl_ptr[r] + rr] = 1.0
            cols.append(case.dense @ m); meta.append((b, combo))
    return np.array(cols), meta


def test_column_generation_is_exact_on_a_tiny_instance(tiny):
    """'an exact method called column generation': run to termination; the
    terminal objective equals the master solved over ALL 96 deliverable apertures, and no
    aperture has a negative reduced cost."""
    vp = _params(tiny)
    plan = orc.run(tiny, max_apertures=96, master_tol=1e-12, price_tol=1e-9, keep_A=True)
    assert plan.converged
    A_all, _ = _all_apertures(tiny)
    assert A_all.shape[0] == 2 * 48
    full = orc.master(A_all, np.zeros(A_all.shape[0]), vp, tol=1e-12, max_iter=2000)
    ref = minimize(lambda y: _F_numpy(A_all, y, vp), np.full(A_all.shape[0], 0.01),
                   jac=lambda y: _gradF_numpy(A_all, y, vp), bounds=[(0, None)] * A_all.shape[0],
                   method="L-BFGS-B", options={"ftol": 1e-15, "gtol": 1e-12, "maxiter": 20000, "maxfun": 100000})
    assert plan.objective == pytest.approx(full.objective, rel=1e-7)
    assert plan.objective <= ref.fun * (1 + 1e-6)
    # reduced costs of every aperture at the terminal dose
    red = _gradF_numpy(A_all, np.zeros(A_all.shape[0]), vp) * 0 + A_all @ (
        -2 * vp.a * np.maximum(0, vp.tm - plan.y @ plan.A) + 2 * vp.b * np.maximum(0, plan.y @ plan.A - vp.tp))
    assert red.min() >= -1e-7 * np.abs(red).max()


def test_column_generation_history_is_monotone_and_prices_negative(mini):
    plan = orc.run(mini, max_apertures=12, master_tol=1e-11)
    f = [h.objective for h in plan.history]
    assert plan.history[0].objective_before == pytest.approx(10.0, rel=1e-12)   # F(0) = alpha (T^-)^2
    for h in plan.history:
        assert h.price < 0.0
        assert h.objective < h.objective_before        # strict decrease while the price is negative
        assert h.kkt <= 1e-8
    assert all(f[i + 1] < f[i] for i in range(len(f) - 1))
    assert plan.objective == pytest.approx(f[-1], rel=1e-9)     # F(D x(y)) == F(A y)


def test_fmo_lower_bound(tiny):
    """Every aperture plan is a beamlet plan (eq. 7), so F*_DAO(K) >= F*_FMO, with
    equality reachable only at CG termination.  FMO solved by L-BFGS-B on x >= 0."""
    vp = _params(tiny)
    D = tiny.dense
    Fx = lambda x: float(np.sum(vp.a * np.maximum(0, vp.tm - D @ x) ** 2 + vp.b * np.maximum(0, D @ x - vp.tp) ** 2))
    gx = lambda x: D.T @ (-2 * vp.a * np.maximum(0, vp.tm - D @ x) + 2 * vp.b * np.maximum(0, D @ x - vp.tp))
    ref = minimize(Fx, np.full(tiny.n_bl, 0.01), jac=gx, bounds=[(0, None)] * tiny.n_bl, method="L-BFGS-B",
                   options={"ftol": 1e-15, "gtol": 1e-12, "maxiter": 20000})
    for K in (1, 3, 8):
        plan = orc.run(tiny, max_apertures=K, master_tol=1e-11)
        assert plan.objective >= ref.fun * (1 - 1e-9)


def test_cfg0_runs_to_50_apertures_in_seconds(cfg0):
    import time
    t = time.time()
    plan = orc.run(cfg0, max_apertures=50, master_tol=1e-10)
    assert time.time() - t < 60
    assert 1 <= len(plan.beams) <= 50
    assert plan.objective < 1.0 and all(h.kkt < 1e-8 for h in plan.history)


def test_stored_cfg1_plan_is_converged_at_every_iteration():
    """tests/golden/oracle_plan_cfg1.json (written by make_oracle_plan.py from oracle/ only): every master solve of
    the stored free-running plan met the KKT conditions to 1e-8 (absolute, in units of dF/dy; F is 1e-2 .. 1 along
    the plan), no duplicate candidate ever appeared (reading S6 never fired) and the objective fell monotonically."""
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_plan_cfg1.json")) as f:
        gold = json.load(f)
    assert len(gold["kkt"]) == gold["n_apertures"] == 50
    assert max(gold["kkt"]) <= 1e-8
    assert gold["n_duplicates"] == 0 and not gold["stalled"] and not gold["converged"]
    f = np.asarray(gold["master_objective"])
    assert (np.diff(f) < 0).all() and (np.asarray(gold["price"]) < 0).all()
    assert gold["objective"] == pytest.approx(f[-1], rel=1e-9)
