"""GPU parity tests: the CUDA path (through the C ABI / ctypes binding) against the fp64 CPU oracle
on the same seeded inputs.  Tolerances are BASELINE.json's north star:
  * same fp32 w -> leaf positions bit-exact whenever best and second-best differ by > 1e-6 relative;
  * dose and gradient within 1e-4 relative (L-inf, normalised by the prescription dose / max |g|);
  * final 50-aperture objective within 1e-3 relative.
"""
import numpy as np
import pytest

from oracle import dao_oracle as orc
from paper_1003_5402_b200.inputs import phantom
import parity_utils as pu

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
REL_DOSE = 1e-4
REL_OBJ = 1e-3
GP_MAX_ITER = 200000   # iteration cap for master_method 0 (plain gradient projection converges linearly)


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class CsrCase:
    """Random CSR incl. empty rows / columns wrapped as a one-beam 'phantom' for kernel tests."""

    def __init__(self, n_vox, n_bl, density, seed, row_len=None):
        self.row_ptr, self.col_idx, self.val, self.dense = phantom.random_csr(n_vox, n_bl, density, seed)
        self.n_vox, self.n_bl, self.nnz = n_vox, n_bl, int(self.val.size)
        rl = row_len or n_bl
        n_rows = (n_bl + rl - 1) // rl
        self.n_beams, self.n_rows = 1, n_rows
        self.beam_row_ptr = np.array([0, n_rows], np.int32)
        self.row_bl_ptr = np.minimum(np.arange(n_rows + 1) * rl, n_bl).astype(np.int32)
        rng = np.random.default_rng(seed + 100)
        self.vox_struct = rng.integers(-1, 2, n_vox).astype(np.int32)
        self.t_under = np.array([1.0, 0.0], np.float32); self.w_under = np.array([10.0, 0.0], np.float32)
        self.t_over = np.array([1.05, 0.3], np.float32); self.w_over = np.array([5.0, 2.0], np.float32)
        self.prescription = 1.0


# ----------------------------------------------------------------------------- steps 2, 4 (isolated)
@pytest.mark.parametrize("case", ["cfg0", "mini", "csr_small", "csr_ragged", "csr_wide"])
def test_spmv_and_transpose_match_oracle(D, case, cfg0, mini):
    ph = {"cfg0": cfg0, "mini": mini}.get(case)
    if ph is None:
        ph = {"csr_small": lambda: CsrCase(37, 5, 0.4, 1), "csr_ragged": lambda: CsrCase(1031, 77, 0.2, 2),
              "csr_wide": lambda: CsrCase(300, 30000, 0.002, 3, row_len=100)}[case]()
    rng = np.random.default_rng(7)
    x = rng.random(ph.n_bl).astype(np.float32)
    g = rng.standard_normal(ph.n_vox).astype(np.float32)
    for dev_in in (False, True):
        with D.Dao(ph, device_inputs=dev_in) as d:
            z = d.spmv(_dev(x)).cpu().numpy()
            w = d.spmv_t(_dev(g)).cpu().numpy()
    zo = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x.astype(np.float64))
    wo = orc.beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, g.astype(np.float64), ph.n_bl)
    assert np.abs(z - zo).max() <= REL_DOSE * max(np.abs(zo).max(), 1e-30)
    assert np.abs(w - wo).max() <= REL_DOSE * max(np.abs(wo).max(), 1e-30)
    # fp32 storage of an fp64-accumulated sum: in fact within a few ulp
    assert np.abs(z - zo).max() <= 2e-7 * max(np.abs(zo).max(), 1e-30)
    assert np.abs(w - wo).max() <= 2e-7 * max(np.abs(wo).max(), 1e-30)


@pytest.mark.parametrize("sigma", [1, 64, 4096])
def test_spmv_independent_of_sell_window(D, mini, sigma):
    """The internal voxel order (sorting window) must not change any result (row sums are per lane)."""
    x = np.random.default_rng(3).random(mini.n_bl).astype(np.float32)
    with D.Dao(mini, sell_sigma=sigma) as d, D.Dao(mini) as d0:
        assert d.dims().sell_sigma == sigma
        z, z0 = d.spmv(_dev(x)).cpu().numpy(), d0.spmv(_dev(x)).cpu().numpy()
        F, F0 = d.eval_x(_dev(x)), d0.eval_x(_dev(x))
        g, g0 = d.get_vector(D.VEC_G), d0.get_vector(D.VEC_G)
    assert np.array_equal(z, z0) and np.array_equal(g, g0)
    assert abs(F - F0) <= 1e-13 * abs(F0)


# ----------------------------------------------------------------------------- step 3 (fused epilogue)
@pytest.mark.parametrize("case", ["cfg0", "mini", "mini_reopt"])
def test_objective_and_gradient_match_oracle(D, case, cfg0, mini, mini_reopt):
    ph = {"cfg0": cfg0, "mini": mini, "mini_reopt": mini_reopt}[case]
    vp = orc.voxel_params_of(ph)
    rng = np.random.default_rng(11)
    with D.Dao(ph) as d:
        for scale in (0.0, 0.02, 0.05, 0.2):
            x = (scale * rng.random(ph.n_bl)).astype(np.float32)
            F = d.eval_x(_dev(x))
            z, g = d.get_vector(D.VEC_Z), d.get_vector(D.VEC_G)
            zo = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x.astype(np.float64))
            Fo, go = orc.objective(zo, vp), orc.voxel_gradient(zo, vp)
            assert abs(F - Fo) <= 1e-12 * max(Fo, 1e-30)
            assert np.abs(z - zo).max() <= REL_DOSE * ph.prescription
            assert np.abs(g - go).max() <= REL_DOSE * max(np.abs(go).max(), 1e-30)
    if case == "mini_reopt":
        # closed form (PAPER.md:75-83 with alpha = beta = 1): F(z = 0) = sum over target voxels of T_j^2
        t = ph.vox_threshold.astype(np.float64)
        assert abs(orc.objective(np.zeros(ph.n_vox), vp) - float((t[ph.vox_struct == 0] ** 2).sum())) < 1e-9
    else:
        # closed form: F(z = 0) = sum over targets of alpha_s (T_s^-)^2
        assert abs(orc.objective(np.zeros(ph.n_vox), vp) - 10.0) < 1e-12


# ----------------------------------------------------------------------------- steps 5, 6
@pytest.mark.parametrize("n_rows,row_len,seed", [(1000, 20, 0), (1000, 40, 1), (3000, 80, 2), (257, 33, 3), (64, 100, 4)])
def test_pricing_sweep_bit_exact(D, mini, n_rows, row_len, seed):
    w, brp, rbp = phantom.pricing_rows(n_rows, row_len, rows_per_beam=40, seed=seed)
    with D.Dao(mini) as d:
        le, ri, vs, bp, best = d.price_from_w(_dev(w), _dev(rbp), _dev(brp))
        le, ri, vs, bp, best = (t.cpu().numpy() for t in (le, ri, vs, bp, best))
    n_exact, n_band = pu.check_rows(w, rbp, le, ri, vs)
    assert n_exact >= 0.99 * n_rows
    pr = orc.price(w.astype(np.float64), brp, rbp)
    pu.check_beam(bp, best[0], pr.beam_price)


def test_pricing_ties_and_edge_rows(D, mini):
    """Integer-valued rows (exact arithmetic, many exact ties): the fixed tie-break (smallest left
    leaf, then smallest right leaf; closed row wins ties at 0) must match the oracle bit for bit."""
    rng = np.random.default_rng(5)
    rows = [rng.integers(-2, 3, n).astype(np.float32) for n in rng.integers(1, 70, 400)]
    rows += [np.array([2, -3, 1, -2, 4], np.float32),            # tests/golden/row_scan_example.txt
             np.zeros(7, np.float32), np.ones(40, np.float32), -np.ones(65, np.float32),
             np.array([-1], np.float32), np.array([1], np.float32), np.array([0, 0, -1, 0, 0], np.float32),
             np.array([-1, 1, -1, 1, -1], np.float32), np.r_[np.zeros(33), -1, np.zeros(40)].astype(np.float32)]
    rbp = np.r_[0, np.cumsum([r.size for r in rows])].astype(np.int32)
    brp = np.array([0, 100, 250, len(rows)], np.int32)
    w = np.concatenate(rows)
    with D.Dao(mini) as d:
        le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(w), _dev(rbp), _dev(brp)))
    pr = orc.price(w.astype(np.float64), brp, rbp)
    assert np.array_equal(le, pr.left) and np.array_equal(ri, pr.right)
    assert np.array_equal(vs, pr.vstar)
    np.testing.assert_allclose(bp, pr.beam_price, rtol=0, atol=0)
    assert best[0] == pr.best_beam
    k = len(rows) - 9
    assert (le[k], ri[k], vs[k]) == (1, 4, -4.0)


def test_pricing_on_own_tables(D, mini):
    w = np.random.default_rng(9).standard_normal(mini.n_bl).astype(np.float32)
    with D.Dao(mini) as d:
        le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(w)))
    pu.check_rows(w, mini.row_bl_ptr, le, ri, vs)
    pu.check_beam(bp, best[0], orc.price(w.astype(np.float64), mini.beam_row_ptr, mini.row_bl_ptr).beam_price)


# ----------------------------------------------------------------------------- lock-step protocol
@pytest.mark.parametrize("case,n_ap,method", [("cfg0", 12, 2), ("mini", 20, 2), ("mini_reopt", 12, 2),
                                               ("mini", 10, 0), ("mini", 20, 1), ("mini", 20, 3)])
def test_lockstep_against_oracle(D, case, n_ap, method, cfg0, mini, mini_reopt):
    """SURVEY 8(c) lock-step: at every column-generation iteration the oracle recomputes each step
    from the GPU's own state; isolates every step's error from trajectory divergence."""
    ph = {"cfg0": cfg0, "mini": mini, "mini_reopt": mini_reopt}[case]
    # method 0 is the plain gradient projection PAPER.md:134 names: same stopping test, many more iterations
    with D.Dao(ph, k_max=n_ap, master_method=method, master_max_iter=GP_MAX_ITER if method == 0 else 2000) as d:
        for it in range(n_ap):
            info = d.price()
            plan = d.get_plan()
            y = d.get_vector(D.VEC_Y)[:len(plan.beams)]
            lefts = [plan.leaves(k)[0] for k in range(len(plan.beams))]
            rights = [plan.leaves(k)[1] for k in range(len(plan.beams))]
            vp, x_o, z_o, g_o, w_o, F_o = pu.oracle_state_from_plan(ph, plan.beams, lefts, rights, y)
            z, g, w = d.get_vector(D.VEC_Z), d.get_vector(D.VEC_G), d.get_vector(D.VEC_W)
            assert np.abs(z - z_o).max() <= REL_DOSE * ph.prescription
            assert np.abs(g - g_o).max() <= REL_DOSE * np.abs(g_o).max()
            assert np.abs(w - w_o).max() <= REL_DOSE * np.abs(w_o).max()
            assert abs(info.objective - F_o) <= 1e-6 * F_o
            le, ri, vs = d.get_vector(D.VEC_LEFT), d.get_vector(D.VEC_RIGHT), d.get_vector(D.VEC_VSTAR)
            pu.check_rows(w, ph.row_bl_ptr, le, ri, vs)               # oracle prices the GPU's fp32 w
            pr = orc.price(w.astype(np.float64), ph.beam_row_ptr, ph.row_bl_ptr)
            pu.check_beam(d.get_vector(D.VEC_BEAM_PRICE), info.beam, pr.beam_price)
            assert abs(info.price - pr.beam_price[info.beam]) <= 1e-9 * max(1.0, abs(info.price))
            if info.converged:
                break
            m = d.solve_master()
            assert m.n_apertures == it + 1
            plan = d.get_plan()
            lefts = [plan.leaves(k)[0] for k in range(len(plan.beams))]
            rights = [plan.leaves(k)[1] for k in range(len(plan.beams))]
            A = pu.oracle_columns(ph, plan.beams, lefts, rights)
            res = orc.master(A, np.zeros(len(plan.beams)), vp, tol=1e-10)
            rel = (m.objective - res.objective) / res.objective
            assert -1e-5 <= rel <= REL_OBJ, (it, m.objective, res.objective, m.n_pg_iter, m.hit_max_iter)
            # the master's own z equals A y
            yk = d.get_vector(D.VEC_Y)[:len(plan.beams)]
            mz = d.get_vector(D.VEC_MASTER_Z)
            assert np.abs(mz - yk @ A).max() <= 1e-6 * max(1.0, np.abs(mz).max())


@pytest.mark.parametrize("method", [0, 1, 2, 3])
def test_master_on_oracle_pool(D, mini, method):
    """dao_set_pool + dao_resolve_master on the oracle's 15-aperture pool: same optimum value (the optimum is unique,
    PAPER.md:114, whichever of the four methods reaches it; 0 = the gradient projection PAPER.md:134 names)."""
    plan = orc.run(mini, 15, keep_A=True)
    vp = orc.voxel_params(mini.vox_struct, mini.t_under, mini.w_under, mini.t_over, mini.w_over)
    with D.Dao(mini, master_method=method, master_max_iter=GP_MAX_ITER if method == 0 else 2000) as d:
        d.set_pool(plan.beams, plan.lefts, plan.rights)
        m = d.resolve_master()
        y = d.get_vector(D.VEC_Y)[:15]
    assert m.n_apertures == 15 and not m.hit_max_iter
    assert abs(m.objective - plan.objective) <= 1e-5 * plan.objective
    f_chk, grad = orc.master_gradient(plan.A, y, vp)          # KKT of the GPU's y in the oracle's arithmetic
    assert abs(f_chk - m.objective) <= 1e-6 * f_chk      # A is stored in fp32 on the GPU
    assert (grad >= -1e-5 * max(1.0, f_chk)).all()
    assert (np.abs(grad[y > 0]) <= 1e-5 * max(1.0, f_chk)).all()


# ----------------------------------------------------------------------------- free-running plans
@pytest.mark.parametrize("case,method,n_ap", [("cfg0", 2, 50), ("mini", 2, 50), ("mini_reopt", 2, 50), ("mini", 0, 15),
                                               ("mini", 1, 50), ("mini", 3, 50)])
def test_free_running_50_apertures(D, case, method, n_ap, cfg0, mini, mini_reopt):
    """(15 apertures for method 0: plain gradient projection needs ~1e4-1e5 iterations per solve as the pool grows)"""
    ph = {"cfg0": cfg0, "mini": mini, "mini_reopt": mini_reopt}[case]
    with D.Dao(ph, k_max=n_ap, master_method=method, master_max_iter=GP_MAX_ITER if method == 0 else 2000) as d:
        info = d.run(n_ap)
        plan = d.get_plan()
        hist = d.get_vector(D.VEC_HISTORY)[:info.n_apertures]
    ref = orc.run(ph, n_ap)
    assert info.n_hit_max_iter == 0
    assert abs(info.objective - ref.objective) <= REL_OBJ * ref.objective
    assert abs(plan.objective - info.objective) <= 1e-12 * info.objective
    # monotone decrease of the master optimum (convexity + warm start)
    f = np.r_[hist["objective_before"][:1], hist["objective"]]
    assert (np.diff(f) <= 1e-9 * f[:-1]).all()
    assert (hist["price"] < 0).all()
    assert (plan.intensity >= 0).all()
    n_same = sum(1 for k in range(min(len(ref.beams), len(plan.beams)))
                 if plan.beams[k] == ref.beams[k] and np.array_equal(plan.leaves(k)[0], ref.lefts[k])
                 and np.array_equal(plan.leaves(k)[1], ref.rights[k]))
    print(f"{case}: F_gpu={info.objective:.10g} F_oracle={ref.objective:.10g} same apertures {n_same}/{len(ref.beams)}"
          f" pg iterations {info.n_pg_iter_total}")


def test_run_is_deterministic_and_resettable(D, mini):
    with D.Dao(mini, k_max=12) as d:
        a = d.run(12); pa = d.get_plan(); za = d.get_vector(D.VEC_Z)
        d.reset()
        b = d.run(12); pb = d.get_plan(); zb = d.get_vector(D.VEC_Z)
    assert a.objective == b.objective and np.array_equal(za, zb)
    assert np.array_equal(pa.beams, pb.beams) and np.array_equal(pa.left, pb.left) and np.array_equal(pa.intensity, pb.intensity)


def test_terminates_when_optimal(D, tiny):
    """Tiny instance run to termination: converged flag, non-negative reduced costs in the oracle's
    arithmetic at the GPU's plan, and the oracle's terminal objective."""
    with D.Dao(tiny) as d:
        info = d.run(50)
        plan = d.get_plan()
        y = d.get_vector(D.VEC_Y)[:info.n_apertures]
    ref = orc.run(tiny, 50)
    assert info.converged and ref.converged
    assert abs(info.objective - ref.objective) <= 1e-6 * ref.objective
    lefts = [plan.leaves(k)[0] for k in range(len(plan.beams))]
    rights = [plan.leaves(k)[1] for k in range(len(plan.beams))]
    _, _, _, _, w_o, _ = pu.oracle_state_from_plan(tiny, plan.beams, lefts, rights, y)
    pr = orc.price(w_o, tiny.beam_row_ptr, tiny.row_bl_ptr)
    assert pr.price >= -1e-5


# ----------------------------------------------------------------------------- errors
def test_error_paths(D, tiny):
    import copy
    bad = copy.copy(tiny); bad.row_ptr = tiny.row_ptr.copy(); bad.row_ptr[3] = bad.row_ptr[4] + 1
    with pytest.raises(D.DaoError) as e:
        D.Dao(bad)
    assert e.value.status == 2
    bad = copy.copy(tiny); bad.col_idx = tiny.col_idx.copy(); bad.col_idx[5] = tiny.n_bl
    with pytest.raises(D.DaoError) as e:
        D.Dao(bad)
    assert e.value.status == 2
    bad = copy.copy(tiny); bad.val = tiny.val.copy(); bad.val[0] = np.nan
    with pytest.raises(D.DaoError) as e:
        D.Dao(bad)
    assert e.value.status == 1
    with pytest.raises(D.DaoError) as e:
        D.Dao(tiny, k_max=D.MAX_APERTURES + 1)
    assert e.value.status == 6
    with D.Dao(tiny, k_max=2) as d:
        with pytest.raises(D.DaoError) as e:
            d.solve_master()                      # no pending candidate
        assert e.value.status == 5
        with pytest.raises(D.DaoError):
            d.run(3)                              # > k_max
        d.price(); d.solve_master(); d.price(); d.solve_master()
        info = d.price()                          # pool full: no candidate is stored
        with pytest.raises(D.DaoError) as e:
            d.solve_master()
        assert e.value.status == 5
        assert d.get_plan().beams.size == 2
