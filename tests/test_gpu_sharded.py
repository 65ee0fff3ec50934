"""GPU parity of the voxel-row sharding slice (paper_1003_5402_b200/sharded.py): R slab contexts on
ONE GPU, run one after the other (kernels of different ranks never wait on one another), their shares added in
rank order on the host -- against the fp64 oracle on the whole problem and against the unsharded context.

What is checked per slab count R: the slab's share of F with |v_s| of the WHOLE problem (dao_structs.struct_count,
eq. 9-10), the partial sums of w = D^T pi (eq. 8), and that pricing on the summed gradient takes the decision of the
unsharded path.
"""
import numpy as np
import pytest

from oracle import dao_oracle as orc
from paper_1003_5402_b200 import sharded

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


def _check(D, ph, world, seed):
    rng = np.random.default_rng(seed)
    x = (0.05 * rng.random(ph.n_bl)).astype(np.float32)
    xd = torch.from_numpy(x).cuda()
    # the oracle on the whole problem
    vp = orc.voxel_params_of(ph)
    zo = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x.astype(np.float64))
    Fo, go = orc.objective(zo, vp), orc.voxel_gradient(zo, vp)
    wo = orc.beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, go, ph.n_bl)
    # the unsharded context
    with D.Dao(ph, k_max=4) as d:
        F1 = d.eval_x(xd)
        g1 = d.get_vector(D.VEC_G)
        w1 = d.spmv_t(torch.from_numpy(g1).cuda()).cpu().numpy()
        le1, ri1, _, bp1, best1 = (t.cpu().numpy() for t in d.price_from_w(torch.from_numpy(w1).cuda()))
    # R slabs, one after the other
    f_parts, w_parts, g_parts, last = [], [], [], None
    for rank in range(world):
        it = sharded.ShardedIteration(D, ph, rank, world, k_max=4)
        try:
            f_r, w_r = it.local_shares(xd)
            f_parts.append(f_r); w_parts.append(w_r); g_parts.append(it.ctx.get_vector(D.VEC_G))
            if rank == world - 1:
                w_sum = sharded.sum_in_rank_order(w_parts)
                last = [t.cpu().numpy() for t in it.price(w_sum)]
        finally:
            it.close()
    F = float(np.sum(f_parts))
    g = np.concatenate(g_parts)
    w = sharded.sum_in_rank_order(w_parts)
    assert g.size == ph.n_vox
    assert abs(F - Fo) <= 1e-10 * Fo and abs(F - F1) <= 1e-12 * F1          # shares of F with the global |v_s|
    assert np.abs(g - go).max() <= 1e-4 * np.abs(go).max() and np.array_equal(g, g1)   # pi is local: same bits
    assert np.abs(w - wo).max() <= 2e-7 * np.abs(wo).max() + 1e-4 * 0            # north star: 1e-4; measured: fp32 rounding
    assert np.abs(w - w1).max() <= 2e-7 * np.abs(w1).max()
    # replicated pricing on the summed gradient: the decision of the unsharded path
    le, ri, _, bp, best = last
    assert int(best[0]) == int(best1[0])
    assert np.allclose(bp, bp1, rtol=1e-6, atol=1e-6 * np.abs(bp1).max())
    b = int(best[0])
    rows = slice(ph.beam_row_ptr[b], ph.beam_row_ptr[b + 1])
    same = np.mean((le[rows] == le1[rows]) & (ri[rows] == ri1[rows]))
    assert same >= 0.9                      # leaves may differ only where two intervals tie to fp32 rounding of w
    return F, float(np.abs(w - wo).max() / np.abs(wo).max())


@pytest.mark.parametrize("world", [1, 2, 3])
def test_sharded_iteration_matches_oracle_on_mini(D, mini, world):
    _check(D, mini, world, seed=11)


def test_sharded_iteration_reoptimisation_mode(D, mini_reopt):
    """Per-voxel thresholds travel with the slab; weights are not divided by |v_s| in this mode."""
    _check(D, mini_reopt, 2, seed=12)


def test_sharded_iteration_at_full_size(D):
    """configs[1] (603,844 voxels, 47.2M non-zeros) over 4 slabs balanced by non-zeros."""
    from paper_1003_5402_b200.inputs import phantom
    ph = phantom.make("cfg1", seed=0)
    F, err = _check(D, ph, 4, seed=13)
    nnz = [int(ph.row_ptr[v1] - ph.row_ptr[v0]) for v0, v1 in sharded.slab_bounds(ph.n_vox, 4, ph.row_ptr)]
    assert max(nnz) - min(nnz) <= 4 * int(np.diff(ph.row_ptr).max())
    print(f"cfg1 over 4 slabs: F={F:.10g}, |w - w_oracle|/max|w| = {err:.2e}, non-zeros per slab {nnz}")
