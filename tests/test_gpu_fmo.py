"""GPU parity of the FMO workload: min_{x >= 0} F(D x) by projected
gradient on the device (dao_fmo_solve) against the oracle's FMO optimum.  The optimum VALUE is unique
(convex), x need not be: parity is on F (north star: 1e-3), and on the KKT conditions evaluated by the
oracle at the GPU's x."""
import json
import os

import numpy as np
import pytest

from oracle import dao_oracle as orc
from paper_1003_5402_b200.inputs import phantom

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
REL_OBJ = 1e-3
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


def _oracle_at(ph, x):
    """F, w and the first-order optimality gap of the oracle at beamlet intensities x."""
    vp = orc.voxel_params_of(ph)
    z = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x.astype(np.float64))
    g = orc.voxel_gradient(z, vp)
    w = orc.beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, g, ph.n_bl)
    # convexity: F(x) - F* <= w.(x - x*) <= w.x + max(0, -min w) |x*|_1, with |x*|_1 taken as 2 |x|_1
    gap = float(w @ x) + max(0.0, -float(w.min())) * 2.0 * float(x.sum())
    return orc.objective(z, vp), z, w, gap


@pytest.mark.parametrize("case", ["tiny", "cfg0"])
def test_fmo_matches_oracle_optimum(D, case, tiny, cfg0):
    ph = {"tiny": tiny, "cfg0": cfg0}[case]
    ref = orc.fmo(ph, method="newton", tol=1e-10)
    with D.Dao(ph) as d:
        info = d.fmo_solve(max_iter=20000, tol=1e-7)
        x = d.get_vector(D.VEC_X).astype(np.float64)
        z = d.get_vector(D.VEC_Z)
    rel = (info.objective - ref.objective) / ref.objective
    assert -1e-6 <= rel <= REL_OBJ, (info.objective, ref.objective, info.n_iter, info.converged)
    assert (x >= 0).all()
    F_o, z_o, w_o, gap = _oracle_at(ph, x)
    assert abs(F_o - info.objective) <= 1e-6 * F_o
    assert np.abs(z - z_o).max() <= 1e-4 * ph.prescription
    assert gap <= REL_OBJ * F_o
    print(f"{case}: F_gpu={info.objective:.10g} F_oracle={ref.objective:.10g} rel={rel:.2e} iters={info.n_iter} "
          f"ls={info.n_ls_evals} restarts={info.n_restarts} converged={info.converged}")


def test_fmo_mini_properties_and_dao_lower_bound(D, mini):
    """mini (241 beamlets): the dense-Newton oracle takes minutes, so its optimum is a stored fixture
    (tests/golden/oracle_fmo_mini.json); plus properties the oracle evaluates at the GPU's x: same
    objective, first-order optimality gap within 1e-3, and the lower-bound relation of eq. 7 against the GPU's own 50-aperture DAO plan."""
    with open(os.path.join(GOLDEN, "oracle_fmo_mini.json")) as f:
        gold = json.load(f)
    assert (gold["n_vox"], gold["n_bl"], gold["nnz"]) == (mini.n_vox, mini.n_bl, mini.nnz)
    with D.Dao(mini) as d:
        info = d.fmo_solve(max_iter=5000, tol=1e-6)
        x = d.get_vector(D.VEC_X).astype(np.float64)
        a = d.fmo_solve(max_iter=5000, tol=1e-6)                      # from x = 0 again: bit-reproducible
        xa = d.get_vector(D.VEC_X).astype(np.float64)
        plan = d.run(50)
    assert a.objective == info.objective and a.n_iter == info.n_iter and np.array_equal(x, xa)
    rel = (info.objective - gold["objective"]) / gold["objective"]
    assert -1e-6 <= rel <= REL_OBJ, (info.objective, gold["objective"], info.n_iter)
    F_o, _, _, gap = _oracle_at(mini, x)
    assert abs(F_o - info.objective) <= 1e-6 * F_o
    assert gap <= REL_OBJ * F_o, (gap, F_o, info.n_iter)
    assert info.objective <= plan.objective * (1 + 1e-6)
    pg = orc.fmo(mini, method="pg", tol=1e-4, max_iter=300)           # plain PG oracle: an upper bound of F*
    assert info.objective <= pg.objective * (1 + 1e-6)
    print(f"mini: F_fmo={info.objective:.10g} (gap {gap:.2e}, {info.n_iter} iterations) F_dao50={plan.objective:.10g} "
          f"F_oracle_pg300={pg.objective:.10g}")


def test_fmo_warm_start_and_iteration_cap(D, mini):
    with D.Dao(mini) as d:
        a = d.fmo_solve(max_iter=30, tol=1e-9)
        assert a.hit_max_iter and a.n_iter == 30 and not a.converged
        b = d.fmo_solve(max_iter=30, tol=1e-9, warm_start=True)
        assert b.objective < a.objective
        c = d.fmo_solve(max_iter=0, tol=1e-9, warm_start=True)        # evaluation only
        assert c.n_iter == 0 and abs(c.objective - b.objective) <= 1e-12 * b.objective
        z0 = d.fmo_solve(max_iter=0)                                  # x = 0: F(0) = alpha (T^-)^2 = 10
        assert abs(z0.objective - 10.0) < 1e-9


def test_fmo_cfg1_full_size(D):
    """configs[1] at full size: the oracle evaluates the GPU's x (objective, optimality gap); F*_FMO must
    lie below the oracle's 50-aperture DAO objective (stored fixture)."""
    ph = phantom.make("cfg1", seed=0)
    with open(os.path.join(GOLDEN, "oracle_plan_cfg1.json")) as f:
        gold = json.load(f)
    with D.Dao(ph) as d:
        first = d.fmo_solve(max_iter=500, tol=1e-6)
        mid = d.fmo_solve(max_iter=2500, tol=1e-6, warm_start=True)
        x_mid = d.get_vector(D.VEC_X).astype(np.float64)
        info = d.fmo_solve(max_iter=5000, tol=1e-6, warm_start=True)
        x = d.get_vector(D.VEC_X).astype(np.float64)
    F_mid, _, _, gap_mid = _oracle_at(ph, x_mid)
    F_o, _, _, gap = _oracle_at(ph, x)
    assert abs(F_o - info.objective) <= 1e-6 * F_o and abs(F_mid - mid.objective) <= 1e-6 * F_mid
    assert (x >= 0).all() and info.objective < mid.objective < first.objective < 10.0
    assert info.objective <= gold["objective"]
    # First-order optimality gap (a rigorous but loose bound: |x*|_1 is taken as 2 |x|_1), evaluated by the oracle.
    # Plain gradient projection over 4,337 beamlets converges slowly: measured on B200, gap / F = 0.44 after 3,000
    # iterations, 0.135 after 8,000, 0.067 after 18,000, 0.026 after 38,000, 0.014 after 78,000 (F = 0.0058678
    # there, 1.6e-4 below the 38,000-iteration value) -- the 1e-3 the small cases reach is out of reach at this size
    # within seconds, so what is asserted is the decay: the bound shrinks and is below 0.2 F after 8,000 iterations.
    assert gap < 0.5 * gap_mid and gap <= 0.2 * F_o, (gap_mid, gap, F_o)
    # F - gap is a lower bound of F*_FMO, and F*_FMO is a lower bound of every aperture plan (eq. 7):
    # the bound computed at either iterate must lie below the later iterate's objective and below the oracle's own
    # 50-aperture DAO objective -- a gap that was too small (a dropped term, a wrong sign) would break the bracket
    assert F_mid - gap_mid <= F_o and F_o - gap <= gold["objective"]
    assert max(F_mid - gap_mid, F_o - gap) <= min(F_o, gold["objective"])
    print(f"cfg1: F_fmo(8000)={info.objective:.10g} gap={gap:.2e} ({gap / F_o:.2e} F); after 3000: F={mid.objective:.10g} gap={gap_mid:.2e}; "
          f"ls={info.n_ls_evals} converged={info.converged} seconds={info.seconds:.3f} F_dao50(oracle)={gold['objective']:.10g}")
