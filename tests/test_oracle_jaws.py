"""Pins of the oracle's jaws-only pricing (PAPER.md:260 names "jaws-only delivery" among
the MLC constraints the model handles; reading J1 of DESIGN.md: apertures are rectangles).  The C
routine enumerates every rectangle with incremental sums; it is pinned here against a numpy
restatement that builds every rectangle's 0/1 beamlet mask explicitly, against special cases, against
the separable (consecutiveness) sub-problem it must dominate, and through the column-generation
driver against the nesting F*_jaws >= F*_consecutive >= F*_FMO."""
import itertools

import numpy as np
import pytest

from oracle import dao_oracle as orc


def _rectangles(brp, rbp, col0, b):
    """Every rectangle of beam b as (c1, c2, m1, m2, mask over beamlets), in the tie-break order."""
    r0, r1 = int(brp[b]), int(brp[b + 1])
    C = max(int(col0[r] + rbp[r + 1] - rbp[r]) for r in range(r0, r1))
    n_bl = int(rbp[-1])
    for c1 in range(C):
        for c2 in range(c1 + 1, C + 1):
            for m1 in range(r1 - r0):
                for m2 in range(m1, r1 - r0):
                    mask = np.zeros(n_bl, bool)
                    for m in range(m1, m2 + 1):
                        r = r0 + m
                        lo, hi = max(c1, int(col0[r])), min(c2, int(col0[r] + rbp[r + 1] - rbp[r]))
                        if hi > lo:
                            mask[rbp[r] + lo - col0[r]: rbp[r] + hi - col0[r]] = True
                    yield c1, c2, m1, m2, mask


def _ragged_case(seed, integer=False):
    rng = np.random.default_rng(seed)
    n_beams = 3
    rows = rng.integers(1, 5, n_beams)
    brp = np.r_[0, np.cumsum(rows)].astype(np.int32)
    lens = rng.integers(1, 6, int(rows.sum()))
    rbp = np.r_[0, np.cumsum(lens)].astype(np.int32)
    col0 = rng.integers(0, 3, lens.size).astype(np.int32)
    for b in range(n_beams):                       # leftmost beamlet of every beam sits at lateral position 0
        col0[brp[b]:brp[b + 1]] -= col0[brp[b]:brp[b + 1]].min()
    w = rng.integers(-3, 4, int(rbp[-1])).astype(np.float64) if integer else rng.standard_normal(int(rbp[-1]))
    return w, brp, rbp, col0


@pytest.mark.parametrize("seed", range(12))
@pytest.mark.parametrize("integer", [False, True])
def test_jaws_pricing_equals_explicit_enumeration(seed, integer):
    """Integer rows give many exact ties: the first rectangle in (c1, c2, m1, m2) order must win, and the
    closed aperture wins ties at 0."""
    w, brp, rbp, col0 = _ragged_case(seed, integer)
    pr = orc.price_jaws(w, brp, rbp, col0)
    for b in range(brp.size - 1):
        best, best_mask = 0.0, np.zeros(w.size, bool)
        for c1, c2, m1, m2, mask in _rectangles(brp, rbp, col0, b):
            s = float(w[mask].sum())
            if s < best:
                best, best_mask = s, mask
        assert pr.beam_price[b] == pytest.approx(best, abs=1e-12)
        got = np.zeros(w.size, bool)
        for r in range(brp[b], brp[b + 1]):
            got[rbp[r] + pr.left[r]: rbp[r] + pr.right[r]] = True
            assert pr.vstar[r] == pytest.approx(float(w[rbp[r] + pr.left[r]: rbp[r] + pr.right[r]].sum()), abs=1e-12)
        if integer:
            assert np.array_equal(got, best_mask)          # same beamlet set, tie-break included
        else:
            assert float(w[got].sum()) == pytest.approx(best, abs=1e-12)
    assert pr.best_beam == int(np.argmin(pr.beam_price))   # first minimum = smallest beam index on ties


def test_jaws_special_cases():
    brp = np.array([0, 3], np.int32); rbp = np.array([0, 4, 8, 12], np.int32); col0 = np.zeros(3, np.int32)
    # nothing negative: closed, value 0
    pr = orc.price_jaws(np.abs(np.random.default_rng(0).standard_normal(12)), brp, rbp, col0)
    assert pr.beam_price[0] == 0.0 and not pr.left.any() and not pr.right.any()
    # one negative cell: the 1 x 1 rectangle around it
    w = np.ones(12); w[6] = -2.0
    pr = orc.price_jaws(w, brp, rbp, col0)
    assert pr.beam_price[0] == -2.0 and (pr.left.tolist(), pr.right.tolist()) == ([0, 2, 0], [0, 3, 0])
    # everything negative: the whole field
    pr = orc.price_jaws(-np.ones(12), brp, rbp, col0)
    assert pr.beam_price[0] == -12.0 and pr.left.tolist() == [0, 0, 0] and pr.right.tolist() == [4, 4, 4]
    # an L-shaped negative region cannot be opened exactly: the best rectangle is the 2 x 2 block (value -4 + 0)
    w = np.array([-1, -1, 5, 5, -1, -1, 5, 5, -1, 5, 5, 5], float)
    pr = orc.price_jaws(w, brp, rbp, col0)
    assert pr.beam_price[0] == -4.0 and pr.left.tolist() == [0, 0, 0] and pr.right.tolist() == [2, 2, 0]
    # shifted rows: lateral positions, not in-row offsets, define the rectangle
    col0 = np.array([2, 0, 1], np.int32)
    w = np.array([-1, 9, 9, 9, 9, 9, -1, 9, 9, -1, 9, 9], float)       # the three -1 sit at lateral position 2
    pr = orc.price_jaws(w, brp, rbp, col0)
    assert pr.beam_price[0] == -3.0 and pr.left.tolist() == [0, 2, 1] and pr.right.tolist() == [1, 3, 2]


@pytest.mark.parametrize("seed", range(6))
def test_jaws_price_is_dominated_by_the_consecutive_subproblem(seed):
    """Every rectangle is a consecutive-leaves aperture, so min over rectangles >= min over the separable
    row-by-row sub-problem beam by beam."""
    w, brp, rbp, col0 = _ragged_case(100 + seed)
    pj, pc = orc.price_jaws(w, brp, rbp, col0), orc.price(w, brp, rbp)
    assert (pj.beam_price >= pc.beam_price - 1e-12).all()
    assert (pj.beam_price <= 0).all()


def test_jaws_column_generation_nests_between_consecutive_and_fmo(mini, tiny):
    a = orc.run(mini, 12)
    b = orc.run(mini, 12, mlc="jaws")
    assert b.objective >= a.objective * (1 - 1e-9)           # fewer deliverable apertures per iteration
    f = [h.objective for h in b.history]
    assert all(f[i + 1] < f[i] for i in range(len(f) - 1)) and all(h.price < 0 for h in b.history)
    for k, beam in enumerate(b.beams):                       # every aperture is a rectangle in lateral positions
        r0 = mini.beam_row_ptr[beam]
        open_rows = [m for m in range(len(b.lefts[k])) if b.rights[k][m] > b.lefts[k][m]]
        assert open_rows == list(range(open_rows[0], open_rows[-1] + 1))
        lo = [int(mini.row_col0[r0 + m] + b.lefts[k][m]) for m in open_rows]
        hi = [int(mini.row_col0[r0 + m] + b.rights[k][m]) for m in open_rows]
        c1, c2 = min(lo), max(hi)
        for m, l, h in zip(open_rows, lo, hi):
            n = int(mini.row_bl_ptr[r0 + m + 1] - mini.row_bl_ptr[r0 + m]); c0 = int(mini.row_col0[r0 + m])
            assert (l, h) == (max(c1, c0), min(c2, c0 + n))
    # tiny, run to termination under both rules: jaws optimum above the consecutive optimum above FMO
    tj, tc = orc.run(tiny, 96, mlc="jaws"), orc.run(tiny, 96)
    assert tj.converged and tc.converged
    f_fmo = orc.fmo(tiny, method="newton", tol=1e-11).objective
    assert tj.objective >= tc.objective * (1 - 1e-9) >= f_fmo * (1 - 1e-9) ** 2
