"""dao_run with and without its per-class event timers.

With ``options.timers = 0`` (the setting bench.py times) dao_run takes another branch: the state block is copied
behind the master, the NEXT iteration's dose SpMV (steps 1-3) is enqueued speculatively behind that copy and the host
waits for the copy's event only; a stalled iteration (reading S6) must throw the speculative dose away because the
re-solve changes x.  Both settings issue the same kernels on the same data in the same order, so everything a run
returns -- apertures, leaves, intensities, objective, the per-iteration history, the counters -- must be IDENTICAL,
for every master method (0 and 1 recompute x with k_intensity, 2 and 3 have the master publish it).  The timers = 1
side is the one the parity tests compare with the oracle (the column-generation loop)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

INFO_FIELDS = ("n_apertures", "n_iterations", "converged", "stalled", "n_duplicates", "n_pg_iter_total", "objective",
               "n_passes_total", "n_hit_max_iter")


@pytest.fixture(scope="module")
def D():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5402_b200 import dao
    dao.load_library()
    return dao


def _run(D, ph, n_ap, **opt):
    with D.Dao(ph, k_max=n_ap, **opt) as d:
        info = d.run(n_ap)
        plan = d.get_plan()
        out = dict(info={f: getattr(info, f) for f in INFO_FIELDS}, plan=plan,
                   hist=d.get_vector(D.VEC_HISTORY)[:info.n_apertures].copy(),
                   y=d.get_vector(D.VEC_Y)[:info.n_apertures].copy(), z=d.get_vector(D.VEC_Z).copy(),
                   x=d.get_vector(D.VEC_X).copy(), launches=info.n_kernel_launches, seconds=info.seconds_master,
                   classes=np.array([info.seconds_intensity, info.seconds_spmv, info.seconds_spmv_t, info.seconds_price,
                                     info.seconds_column, info.seconds_master]),
                   rows=d.get_vector(D.VEC_ITER_SECONDS).reshape(-1, 6).copy())
        # a second run on the same context after a reset must repeat the first (no state left behind by the
        # speculative dose)
        d.reset()
        info2 = d.run(n_ap)
        out["info_again"] = {f: getattr(info2, f) for f in INFO_FIELDS}
    return out


def _same(a, b, same_launches=True):
    assert a["info"] == b["info"], (a["info"], b["info"])
    assert a["info"] == a["info_again"] and b["info"] == b["info_again"]
    pa, pb = a["plan"], b["plan"]
    for f in ("beams", "intensity", "ap_row_ptr", "left", "right"):
        assert np.array_equal(getattr(pa, f), getattr(pb, f)), f
    assert pa.objective == pb.objective
    assert a["hist"].tobytes() == b["hist"].tobytes()
    for f in ("y", "z", "x"):
        assert np.array_equal(a[f], b[f]), f
    if same_launches:
        assert a["launches"] == b["launches"]
    assert a["seconds"] > 0.0 and b["seconds"] == 0.0          # the timers really were on / off
    # DAO_VEC_ITER_SECONDS: one row per aperture added (it pairs with the history records), nothing beyond, the rows
    # never exceed the per-class totals (iterations that added nothing are only in the totals), zeros without timers
    n = a["info"]["n_apertures"]
    assert (a["rows"][:n, 1:] > 0.0).all() and not a["rows"][n:].any() and not b["rows"].any()
    assert (a["rows"].sum(0) <= a["classes"] * (1 + 1e-9) + 1e-12).all()


@pytest.mark.parametrize("method", [0, 1, 2, 3])
def test_plan_is_identical_without_timers(D, mini, method):
    n_ap = 12 if method == 0 else 25                            # plain gradient projection is slow by design
    a = _run(D, mini, n_ap, master_method=method, timers=1)
    b = _run(D, mini, n_ap, master_method=method, timers=0)
    _same(a, b)
    assert a["info"]["n_apertures"] == n_ap
    assert np.allclose(a["rows"].sum(0), a["classes"], rtol=1e-9, atol=1e-12)      # every iteration added an aperture
    # x of the returned plan is the one of eq. (7) whichever kernel wrote it
    plan, x = a["plan"], np.zeros(mini.n_bl)
    for k, bm in enumerate(plan.beams):
        le, ri = plan.leaves(k)
        for m, r in enumerate(range(mini.beam_row_ptr[bm], mini.beam_row_ptr[bm + 1])):
            x[mini.row_bl_ptr[r] + le[m]: mini.row_bl_ptr[r] + ri[m]] += a["y"][k]
    assert np.abs(a["x"] - x).max() <= 1e-6 * max(x.max(), 1e-30)


@pytest.mark.parametrize("method", [0, 1, 2, 3])
@pytest.mark.parametrize("tol", [0.1, 0.03])
def test_converged_on_a_duplicate_without_timers(D, tiny, tol, method):
    """The run that ends on a duplicate candidate after a converged master (S6): the speculative dose is the final one."""
    a = _run(D, tiny, 30, master_method=method, master_tol=tol, timers=1)
    b = _run(D, tiny, 30, master_method=method, master_tol=tol, timers=0)
    _same(a, b)
    assert a["info"]["converged"] == 1 and a["info"]["n_duplicates"] == 1


@pytest.mark.parametrize("method", [0, 1, 2, 3])
def test_stalled_run_without_timers(D, tiny, method):
    """master_max_iter = 0: every master solve stops at once, pricing returns the pool's own aperture with an improving
    price -> two re-solves, then stalled.  The re-solve path discards the speculative dose."""
    a = _run(D, tiny, 30, master_method=method, master_max_iter=0, timers=1)
    b = _run(D, tiny, 30, master_method=method, master_max_iter=0, timers=0)
    _same(a, b, same_launches=False)           # the discarded speculative dose is launched again after the re-solve
    assert b["launches"] > a["launches"]
    # the two re-solves are master time of the call although they add no aperture (and hence no row)
    assert a["classes"][5] > a["rows"][:, 5].sum()
    assert a["info"]["stalled"] == 1 and a["info"]["converged"] == 0 and a["info"]["n_apertures"] == 1
    assert a["info"]["objective"] == pytest.approx(10.0, rel=1e-12)
