"""Pins of the oracle's FMO solver ("the DAO model is the same as the FMO
model ... in which the decision variables are the intensities of all beamlets", solved by "the same
gradient projection method").  orc.fmo(method="pg") is plain gradient projection on the sparse D;
it is pinned against scipy L-BFGS-B, scipy NNLS on the least-squares special case, the KKT
conditions, the dense projected-Newton master on D^T, and the DAO lower-bound relation (eq. 7)."""
import numpy as np
import pytest
from scipy.optimize import minimize, nnls

from oracle import dao_oracle as orc


def _F(D, x, vp):
    z = D @ x
    return float(np.sum(vp.a * np.maximum(0, vp.tm - z) ** 2 + vp.b * np.maximum(0, z - vp.tp) ** 2))


def _grad(D, x, vp):
    z = D @ x
    return D.T @ (-2 * vp.a * np.maximum(0, vp.tm - z) + 2 * vp.b * np.maximum(0, z - vp.tp))


def test_dense_transpose_is_the_transpose(tiny):
    assert np.array_equal(orc.dense_transpose(tiny), tiny.dense.T)


def test_fmo_pg_matches_lbfgsb_newton_and_kkt(tiny):
    vp = orc.voxel_params_of(tiny)
    D = tiny.dense
    ref = minimize(lambda x: _F(D, x, vp), np.full(tiny.n_bl, 0.01), jac=lambda x: _grad(D, x, vp),
                   bounds=[(0, None)] * tiny.n_bl, method="L-BFGS-B",
                   options={"ftol": 1e-15, "gtol": 1e-12, "maxiter": 20000})
    pg = orc.fmo(tiny, method="pg", tol=1e-9, max_iter=200000)
    nt = orc.fmo(tiny, method="newton", tol=1e-11)
    assert pg.objective == pytest.approx(ref.fun, rel=1e-6)
    assert nt.objective == pytest.approx(ref.fun, rel=1e-6)
    assert pg.objective >= nt.objective * (1 - 1e-9)          # nobody beats the optimum
    # KKT in numpy arithmetic at the oracle's x
    g = _grad(D, pg.y, vp)
    assert (pg.y >= 0).all()
    assert g.min() >= -1e-6 * max(1.0, ref.fun)
    assert np.abs(g[pg.y > 0]).max() <= 1e-6 * max(1.0, ref.fun)
    assert pg.kkt <= 1e-6 and _F(D, pg.y, vp) == pytest.approx(pg.objective, rel=1e-12)


def test_fmo_least_squares_special_case_equals_nnls(tiny):
    """T^+ = T^-, beta = alpha on targets and T^+ = 0 on the rest: F is an exact weighted least squares
    (z >= 0 always), whose optimum over x >= 0 is scipy.optimize.nnls's."""
    import copy
    c = copy.copy(tiny)
    c.t_under = np.array([1.0, 0.0], np.float32); c.w_under = np.array([4.0, 0.0], np.float32)
    c.t_over = np.array([1.0, 0.0], np.float32); c.w_over = np.array([4.0, 1.5], np.float32)
    vp = orc.voxel_params_of(c)
    wgt = np.where(c.vox_struct == 0, vp.a, vp.b)
    keep = c.vox_struct >= 0
    M = (np.sqrt(wgt)[:, None] * c.dense)[keep]
    rhs = (np.sqrt(wgt) * np.where(c.vox_struct == 0, 1.0, 0.0))[keep]
    _, rnorm = nnls(M, rhs, maxiter=10000)
    pg = orc.fmo(c, method="pg", tol=1e-10, max_iter=200000)
    assert pg.objective == pytest.approx(rnorm ** 2, rel=1e-6)


def test_fmo_is_a_lower_bound_of_every_dao_plan(tiny):
    """eq. 7: an aperture plan is a beamlet plan, so F*_DAO(K) >= F*_FMO for every K,
    and column generation run to termination on a tiny instance stays above it."""
    f_fmo = orc.fmo(tiny, method="newton", tol=1e-11).objective
    for K in (1, 4, 50):
        plan = orc.run(tiny, max_apertures=K, master_tol=1e-11)
        assert plan.objective >= f_fmo * (1 - 1e-9)


def test_fmo_pg_decreases_monotonically_with_more_iterations(tiny):
    f = [orc.fmo(tiny, method="pg", tol=0.0, max_iter=n).objective for n in (0, 1, 5, 50, 500)]
    vp = orc.voxel_params_of(tiny)
    assert f[0] == pytest.approx(orc.objective(np.zeros(tiny.n_vox), vp), rel=1e-14)      # x = 0
    assert all(f[i + 1] <= f[i] * (1 + 1e-13) for i in range(len(f) - 1)) and f[-1] < f[0]
