"""GPU parity of reading S6 (a candidate that duplicates a pool aperture): the rule of k_price_select / dao_run against
the same rule in the oracle's driver, on the instance where a loose master tolerance forces it to fire."""
import numpy as np
import pytest

from oracle import dao_oracle as orc

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


@pytest.mark.parametrize("method", [0, 1, 2, 3])
@pytest.mark.parametrize("tol", [0.1, 0.03])
def test_duplicate_ends_the_run_as_in_the_oracle(D, tiny, tol, method):
    ref = orc.run(tiny, 30, master_tol=tol)
    assert ref.converged and ref.n_duplicates == 1
    with D.Dao(tiny, k_max=30, master_tol=tol, master_method=method) as d:
        info = d.run(30)
        hist = d.get_vector(D.VEC_HISTORY)[:info.n_apertures]
    assert info.converged == 1 and info.stalled == 0 and info.n_duplicates == 1 and info.n_hit_max_iter == 0
    assert info.n_apertures == len(ref.beams)                      # the same stop iteration under the same rule
    assert info.n_iterations == info.n_apertures + 1               # the last pricing found the duplicate
    # both masters stop anywhere inside the same (loose) tolerance band above the optimum of the pool
    assert abs(info.objective - ref.objective) <= tol * ref.objective
    assert not hist["hit_max_iter"].any()


@pytest.mark.parametrize("method", [0, 1, 2, 3])
def test_duplicate_after_an_unconverged_master_is_reported_as_stalled(D, tiny, method):
    with D.Dao(tiny, k_max=30, master_max_iter=0, master_method=method) as d:
        info = d.run(30)
        pi = d.price()
    assert info.converged == 0 and info.stalled == 1 and info.n_duplicates >= 1 and info.n_hit_max_iter >= 1
    assert info.n_apertures == 1                                   # nothing but the first column could be added
    assert pi.duplicate == 1 and pi.stalled == 1 and pi.converged == 0
    assert info.objective == pytest.approx(10.0, rel=1e-12)        # y = 0 throughout: F(0) = alpha (T^-)^2
