"""Pins of the oracle's pricing under the interdigitation (reading J2) and connectedness (reading J3)
constraints (PAPER.md:260 names them, DESIGN.md states the readings).  The C routine is a
dynamic programme over the leaf rows; it is pinned against exhaustive enumeration of every leaf
configuration of tiny beams (the plain definition), hand cases, and the inclusions between the
feasible sets."""
import itertools

import numpy as np
import pytest

from oracle import dao_oracle as orc


def _states(W):
    return [(a, b) for a in range(W + 1) for b in range(a, W + 1)]


def _feasible(mode, conf):
    """conf: list of (a, b) per row, in lateral positions."""
    if mode == "interdigitation":
        return all(conf[m][0] <= conf[m + 1][1] and conf[m + 1][0] <= conf[m][1] for m in range(len(conf) - 1))
    open_rows = [m for m, (a, b) in enumerate(conf) if a < b]
    if not open_rows:
        return True
    if open_rows != list(range(open_rows[0], open_rows[-1] + 1)):
        return False
    return all(max(conf[m][0], conf[m + 1][0]) < min(conf[m][1], conf[m + 1][1]) for m in open_rows[:-1])


def _brute(mode, w, rbp, col0, r0, r1):
    W = max(int(col0[r] + rbp[r + 1] - rbp[r]) for r in range(r0, r1))
    per_row = []
    for r in range(r0, r1):
        c0, n = int(col0[r]), int(rbp[r + 1] - rbp[r])
        opts = []
        for a, b in _states(W):
            if a < b and (a < c0 or b > c0 + n):
                continue                                    # an open row stays inside its own beamlets
            opts.append((a, b, float(w[rbp[r] + a - c0: rbp[r] + b - c0].sum()) if a < b else 0.0))
        per_row.append(opts)
    best = np.inf
    for conf in itertools.product(*per_row):
        if _feasible(mode, [(a, b) for a, b, _ in conf]):
            best = min(best, sum(v for _, _, v in conf))
    return best


def _case(seed, integer):
    rng = np.random.default_rng(seed)
    rows = rng.integers(1, 4, 2)                            # two beams of 1-3 rows
    brp = np.r_[0, np.cumsum(rows)].astype(np.int32)
    lens = rng.integers(1, 4, int(rows.sum()))
    rbp = np.r_[0, np.cumsum(lens)].astype(np.int32)
    col0 = rng.integers(0, 2, lens.size).astype(np.int32)
    w = rng.integers(-3, 4, int(rbp[-1])).astype(np.float64) if integer else rng.standard_normal(int(rbp[-1]))
    return w, brp, rbp, col0


@pytest.mark.parametrize("mode", ["interdigitation", "connected"])
@pytest.mark.parametrize("seed", range(10))
@pytest.mark.parametrize("integer", [False, True])
def test_chain_pricing_equals_exhaustive_enumeration(mode, seed, integer):
    w, brp, rbp, col0 = _case(seed, integer)
    pr = orc.price_chain(w, brp, rbp, col0, mode)
    for b in range(brp.size - 1):
        r0, r1 = int(brp[b]), int(brp[b + 1])
        assert pr.beam_price[b] == pytest.approx(_brute(mode, w, rbp, col0, r0, r1), abs=1e-12)
        # the returned aperture is feasible and attains the value
        conf = [(int(col0[r] + pr.left[r]), int(col0[r] + pr.right[r])) for r in range(r0, r1)]
        got = sum(float(w[rbp[r] + pr.left[r]: rbp[r] + pr.right[r]].sum()) for r in range(r0, r1))
        assert got == pytest.approx(pr.beam_price[b], abs=1e-12)
        if mode == "connected":
            assert _feasible(mode, conf)
        else:                                               # closed rows are reported as (0, 0): they may park anywhere
            opens = [(m, c) for m, c in enumerate(conf) if c[0] < c[1]]
            for (m0, c0_), (m1, c1_) in zip(opens[:-1], opens[1:]):
                if m1 == m0 + 1:
                    assert c0_[0] <= c1_[1] and c1_[0] <= c0_[1]
    assert pr.best_beam == int(np.argmin(pr.beam_price))


def test_chain_hand_cases():
    brp = np.array([0, 2], np.int32); rbp = np.array([0, 4, 8], np.int32); col0 = np.zeros(2, np.int32)
    # the unconstrained optimum opens [0,1) above [3,4): the left leaf of row 1 would pass the right leaf of row 0
    w = np.array([-1, 5, 5, 5, 5, 5, 5, -1], float)
    assert orc.price(w, brp, rbp).beam_price[0] == -2.0
    assert orc.price_chain(w, brp, rbp, col0, "interdigitation").beam_price[0] == -1.0
    assert orc.price_chain(w, brp, rbp, col0, "connected").beam_price[0] == -1.0
    # touching tips are allowed by the interdigitation rule, but do not make a connected aperture
    w = np.array([-1, -1, 5, 5, 5, 5, -1, -1], float)
    assert orc.price_chain(w, brp, rbp, col0, "interdigitation").beam_price[0] == -4.0
    assert orc.price_chain(w, brp, rbp, col0, "connected").beam_price[0] == -2.0
    # overlapping intervals: all three rules agree with the separable optimum
    w = np.array([5, -1, -1, 5, 5, 5, -1, -1], float)
    for m in ("interdigitation", "connected"):
        assert orc.price_chain(w, brp, rbp, col0, m).beam_price[0] == -4.0
    # a closed row between two open ones: fine for interdigitation (it parks in between), not connected
    brp = np.array([0, 3], np.int32); rbp = np.array([0, 3, 6, 9], np.int32); col0 = np.zeros(3, np.int32)
    w = np.array([-2, -2, -2, 9, 9, 9, -3, -3, -3], float)
    assert orc.price_chain(w, brp, rbp, col0, "interdigitation").beam_price[0] == -15.0
    assert orc.price_chain(w, brp, rbp, col0, "connected").beam_price[0] == -9.0
    # nothing negative: closed
    pr = orc.price_chain(np.ones(9), brp, rbp, col0, "connected")
    assert pr.beam_price[0] == 0.0 and not pr.right.any()


@pytest.mark.parametrize("seed", range(8))
def test_inclusions_between_the_feasible_sets(seed):
    """consecutive >= {interdigitation, connected} always; on a rectangular field also >= jaws-only."""
    rng = np.random.default_rng(50 + seed)
    brp = np.array([0, 4], np.int32); rbp = (np.arange(5) * 5).astype(np.int32); col0 = np.zeros(4, np.int32)
    w = rng.standard_normal(20)
    pc = orc.price(w, brp, rbp).beam_price[0]
    pj = orc.price_jaws(w, brp, rbp, col0).beam_price[0]
    for m in ("interdigitation", "connected"):
        p = orc.price_chain(w, brp, rbp, col0, m).beam_price[0]
        assert pc - 1e-12 <= p <= pj + 1e-12


def test_column_generation_under_the_chain_constraints(mini):
    base = orc.run(mini, 10).objective
    for m in ("interdigitation", "connected"):
        plan = orc.run(mini, 10, mlc=m)
        f = [h.objective for h in plan.history]
        assert all(f[i + 1] < f[i] for i in range(len(f) - 1)) and all(h.price < 0 for h in plan.history)
        assert plan.objective >= base * (1 - 0.05)        # greedy paths differ; the first iteration is identical
        assert plan.history[0].objective == pytest.approx(orc.run(mini, 1).objective, rel=1e-9)
