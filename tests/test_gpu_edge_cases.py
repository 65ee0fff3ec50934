"""Edge cases of the CUDA path: degenerate inputs, maximum pool size, both variants of every kernel that
has two, long leaf rows.  All against the oracle on the same inputs."""
import copy

import numpy as np
import pytest

from oracle import dao_oracle as orc
from paper_1003_5402_b200.inputs import phantom
import parity_utils as pu

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("reserved", [0, 1, 4, 5])
def test_kernel_variants_agree_with_oracle(D, mini, reserved):
    """bit 0: direct-load SpMV instead of the TMA ring; bit 2: span SpMV^T instead of warp-per-row."""
    rng = np.random.default_rng(17)
    x = rng.random(mini.n_bl).astype(np.float32)
    g = rng.standard_normal(mini.n_vox).astype(np.float32)
    with D.Dao(mini, reserved=reserved) as d:
        z = d.spmv(_dev(x)).cpu().numpy()
        w = d.spmv_t(_dev(g)).cpu().numpy()
        info = d.run(6)
    zo = orc.dose(mini.row_ptr, mini.col_idx, mini.val, x.astype(np.float64))
    wo = orc.beamlet_gradient(mini.row_ptr, mini.col_idx, mini.val, g.astype(np.float64), mini.n_bl)
    assert np.abs(z - zo).max() <= 2e-7 * np.abs(zo).max()
    assert np.abs(w - wo).max() <= 2e-7 * np.abs(wo).max()
    ref = orc.run(mini, 6)
    assert abs(info.objective - ref.objective) <= 1e-6 * ref.objective


def test_unpenalised_problem_is_optimal_at_once(D, tiny):
    """No voxel carries a penalty: F = 0, pi = 0, w = 0, pricing proves optimality with an empty pool."""
    c = copy.copy(tiny)
    c.vox_struct = np.full(tiny.n_vox, -1, np.int32)
    with D.Dao(c) as d:
        info = d.price()
        assert info.converged and info.objective == 0.0 and info.price == 0.0
        run = d.run(10)
        assert run.converged and run.n_apertures == 0 and run.objective == 0.0
        assert not d.get_vector(D.VEC_W).any() and not d.get_vector(D.VEC_G).any()
        assert d.get_plan().beams.size == 0


def test_targets_only_overdose_free_start(D, tiny):
    """OAR-only penalties (no target): z = 0 is already optimal (every w_i >= 0 -> all rows stay closed)."""
    c = copy.copy(tiny)
    c.w_under = np.zeros(2, np.float32)
    with D.Dao(c) as d:
        info = d.price()
        le, ri = d.get_vector(D.VEC_LEFT), d.get_vector(D.VEC_RIGHT)
    assert info.converged and info.objective == 0.0
    assert not le.any() and not ri.any()


def test_single_voxel_single_beamlet(D):
    """1 x 1 problem: F(y) = 10 (1 - 0.5 y)^2 on the target voxel -> y* = 2, F* = 0 after one aperture."""
    class One:
        n_vox = n_bl = nnz = n_beams = n_rows = 1
        row_ptr = np.array([0, 1], np.int32); col_idx = np.array([0], np.int32); val = np.array([0.5], np.float32)
        beam_row_ptr = np.array([0, 1], np.int32); row_bl_ptr = np.array([0, 1], np.int32)
        vox_struct = np.array([0], np.int32)
        t_under = np.array([1.0], np.float32); w_under = np.array([10.0], np.float32)
        t_over = np.array([1.05], np.float32); w_over = np.array([5.0], np.float32)
        prescription = 1.0
    with D.Dao(One()) as d:
        first = d.price()
        assert abs(first.objective - 10.0) < 1e-12 and first.beam == 0 and abs(first.price - (-10.0)) < 1e-9
        info = d.run(5)
        plan = d.get_plan()
    assert info.n_apertures == 1 and info.converged and info.objective <= 1e-12
    assert 2.0 - 1e-5 <= plan.intensity[0] <= 2.1 + 1e-5          # any dose in [T^-, T^+] = [1, 1.05] is optimal
    assert plan.leaves(0)[0][0] == 0 and plan.leaves(0)[1][0] == 1


def test_maximum_pool_size(D, mini):
    """k_max = DAO_MAX_APERTURES (128): the run either fills the pool or proves optimality; objective
    against the oracle's."""
    with D.Dao(mini, k_max=D.MAX_APERTURES) as d:
        info = d.run(D.MAX_APERTURES)
        hist = d.get_vector(D.VEC_HISTORY)[:info.n_apertures]
    ref = orc.run(mini, D.MAX_APERTURES)
    assert info.n_apertures == D.MAX_APERTURES or info.converged
    assert abs(info.objective - ref.objective) <= 1e-3 * ref.objective
    f = np.r_[hist["objective_before"][:1], hist["objective"]]
    assert (np.diff(f) <= 1e-9 * f[:-1]).all()
    print(f"k_max=128: {info.n_apertures} apertures, F_gpu={info.objective:.10g} F_oracle={ref.objective:.10g} "
          f"({len(ref.beams)} apertures), pg iterations {info.n_pg_iter_total}")


@pytest.mark.parametrize("row_len", [1, 2, 31, 32, 33, 64, 65, 300, 1000])
def test_pricing_row_lengths_around_the_warp_tiles(D, mini, row_len):
    n_rows = 96
    w, brp, rbp = phantom.pricing_rows(n_rows, row_len, rows_per_beam=7, seed=row_len)
    with D.Dao(mini) as d:
        le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(w), _dev(rbp), _dev(brp)))
    pu.check_rows(w, rbp, le, ri, vs)
    pr = orc.price(w.astype(np.float64), brp, rbp)
    pu.check_beam(bp, best[0], pr.beam_price)
    # integer-valued copy: exact arithmetic, ties everywhere -> bit-exact incl. the tie-break
    wi = np.round(w * 2).astype(np.float32)
    with D.Dao(mini) as d:
        le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(wi), _dev(rbp), _dev(brp)))
    pr = orc.price(wi.astype(np.float64), brp, rbp)
    assert np.array_equal(le, pr.left) and np.array_equal(ri, pr.right) and np.array_equal(vs, pr.vstar)
    assert best[0] == pr.best_beam


@pytest.mark.parametrize("n_rows,row_len", [(32768, 20), (40000, 80), (33001, 88), (33000, 89), (20000, 33)])
def test_pricing_many_rows_thread_per_row_kernel(D, n_rows, row_len):
    """>= 32768 rows of <= 88 beamlets take the thread-per-row kernel (the paper's launch shape);
    longer rows fall back to warp-per-row, decided on the device for caller-provided tables.  Bit-exact on
    integer-valued w (ties), band rule on random w."""
    w, brp, rbp = phantom.pricing_rows(n_rows, row_len, rows_per_beam=40, seed=n_rows % 7)
    wi = np.round(w * 2).astype(np.float32)

    class Host:            # any context whose scratch (>= n_vox entries) holds the caller's tables
        n_vox, n_bl, n_beams, n_rows = 50000, 4, 1, 1
        row_ptr = np.arange(50001, dtype=np.int32); col_idx = (np.arange(50000) % 4).astype(np.int32)
        val = np.ones(50000, np.float32); nnz = 50000
        beam_row_ptr = np.array([0, 1], np.int32); row_bl_ptr = np.array([0, 4], np.int32)
        vox_struct = np.zeros(50000, np.int32)
        t_under = np.array([1.0], np.float32); w_under = np.array([10.0], np.float32)
        t_over = np.array([1.05], np.float32); w_over = np.array([5.0], np.float32)
        prescription = 1.0
    with D.Dao(Host()) as d:
        le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(w), _dev(rbp), _dev(brp)))
        li, rii, vi, bpi, besti = (t.cpu().numpy() for t in d.price_from_w(_dev(wi), _dev(rbp), _dev(brp)))
    pr = orc.price(w.astype(np.float64), brp, rbp)
    assert np.abs(vs - pr.vstar).max() <= 1e-6 * max(1.0, np.abs(pr.vstar).max())
    assert (le == pr.left).mean() >= 0.999 and (ri == pr.right).mean() >= 0.999
    pu.check_beam(bp, best[0], pr.beam_price)
    pi = orc.price(wi.astype(np.float64), brp, rbp)
    assert np.array_equal(li, pi.left) and np.array_equal(rii, pi.right) and np.array_equal(vi, pi.vstar)
    assert besti[0] == pi.best_beam


@pytest.mark.parametrize("mode", ["consecutive", "jaws", "interdigitation", "connected"])
def test_beam_without_leaf_rows(D, tiny, mode):
    """A beam with zero leaf rows offers only the closed aperture: its price is 0 in every MLC mode and it never
    wins against a beam with a negative price (the chain modes once read an unwritten table there)."""
    ph = copy.copy(tiny)
    ph.n_beams = tiny.n_beams + 1
    ph.beam_row_ptr = np.r_[tiny.beam_row_ptr[:1], tiny.beam_row_ptr[:1], tiny.beam_row_ptr[1:]].astype(np.int32)   # beam 0 is empty
    code = {"consecutive": D.MLC_CONSECUTIVE, "jaws": D.MLC_JAWS_ONLY, "interdigitation": D.MLC_INTERDIGITATION,
            "connected": D.MLC_CONNECTED}[mode]
    rng = np.random.default_rng(5)
    with D.Dao(ph, mlc_mode=code, k_max=8) as d:
        for trial in range(3):
            w = rng.standard_normal(ph.n_bl).astype(np.float32) - 0.5
            le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(_dev(w)))
            assert bp[0] == 0.0 and bp[1:].min() < 0.0 and int(best[0]) == 1 + int(np.argmin(bp[1:]))
        info = d.run(8)
        plan = d.get_plan()
    assert info.n_apertures >= 1 and (plan.beams != 0).all()
    ref = orc.run(tiny, 8, mlc=mode)
    assert abs(info.objective - ref.objective) <= 1e-3 * ref.objective      # the empty beam changes nothing


def test_newton_master_at_its_largest_pool(D, mini):
    """master_method = 2 up to 103 apertures (13 block rows of the Hessian; larger k_max falls back to method 1):
    k_max = 100 on mini against the oracle's plan, and both methods against each other."""
    ref = orc.run(mini, 100)
    out = {}
    for method in (1, 2):
        with D.Dao(mini, k_max=100, master_method=method) as d:
            info = d.run(100)
            out[method] = info
    for info in out.values():
        assert info.n_apertures == len(ref.beams) and bool(info.converged) == ref.converged
        assert abs(info.objective - ref.objective) <= 1e-3 * ref.objective
    assert out[2].n_passes_total < out[1].n_passes_total / 5
    print(f"mini k_max=100: {out[2].n_apertures} apertures, F m1={out[1].objective:.10g} m2={out[2].objective:.10g} oracle={ref.objective:.10g}; "
          f"passes over A: {out[1].n_passes_total} (method 1) vs {out[2].n_passes_total} (method 2)")
