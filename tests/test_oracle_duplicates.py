"""Reading S6 of DESIGN.md in the oracle's driver (the paper is silent on a candidate that is already in the pool):
an under-converged master solve leaves a pool aperture with a negative reduced cost, pricing returns that aperture
again, and the loop must stop -- `converged` when the master met its stopping test and its KKT residual explains the
price, `stalled` otherwise -- instead of appending the same column for ever.  Pins on a tiny instance where the
rule is forced to fire by a loose master tolerance / a one-iteration master."""
import numpy as np
import pytest

from oracle import dao_oracle as orc


def _apertures(plan):
    return [(int(b), tuple(map(int, l)), tuple(map(int, r))) for b, l, r in zip(plan.beams, plan.lefts, plan.rights)]


@pytest.mark.parametrize("tol", [0.1, 0.03])
def test_duplicate_after_a_converged_master_ends_the_loop(tiny, tol):
    on = orc.run(tiny, 30, master_tol=tol, keep_A=True)
    off = orc.run(tiny, 30, master_tol=tol, stop_on_duplicate=False)
    assert on.converged and not on.stalled and on.n_duplicates == 1 and len(on.beams) < 30
    # without the rule the same pool is re-extended with copies of its own apertures and never improves
    assert len(off.beams) == 30 and not off.converged
    assert set(_apertures(off)) == set(_apertures(on))
    assert off.objective == pytest.approx(on.objective, rel=1e-12)
    # the objective reported is the (loosely solved) master's over that pool: a tight solve of the SAME pool can
    # only be lower, by less than the tolerance allows, and the exact column-generation optimum lower still
    vp = orc.voxel_params_of(tiny)
    tight = orc.master(on.A, on.y, vp, tol=1e-12)
    exact = orc.run(tiny, 96, master_tol=1e-12)
    assert exact.converged and exact.n_duplicates == 0
    assert exact.objective <= tight.objective * (1 + 1e-9) <= on.objective * (1 + 1e-9)
    assert on.objective - tight.objective <= tol * on.objective
    # the residue bound of the rule: the duplicate's price is negative and explained by the KKT residual of the
    # last master solve (price = dF/dy_k of that aperture)
    f, grad = orc.master_gradient(on.A, on.y, vp)
    assert f == pytest.approx(on.objective, rel=1e-12)
    assert grad.min() < 0 and -grad.min() <= 10 * on.history[-1].kkt


def test_duplicate_after_an_unconverged_master_is_stalled_not_optimal(tiny):
    p = orc.run(tiny, 30, master_tol=1e-10, master_max_iter=1)
    assert p.stalled and not p.converged and p.n_duplicates == 1 and len(p.beams) < 30
    assert p.history[-1].n_master_iter == 1
    exact = orc.run(tiny, 96, master_tol=1e-12)
    assert p.objective > exact.objective * (1 + 1e-3)          # far from optimal: claiming optimality would be wrong


def test_rule_never_fires_at_the_default_tolerances(tiny, mini):
    for ph, n in ((tiny, 96), (mini, 12)):
        p = orc.run(ph, n)
        assert p.n_duplicates == 0 and not p.stalled
