"""Pins for the oracle's dose, objective, gradients and pricing (O1-O7 of DESIGN.md).

Every check compares the oracle with something other than itself: dense numpy products, closed
forms, hand-worked fixtures (tests/golden), finite differences, exhaustive enumeration.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import dao_oracle as orc
from paper_1003_5402_b200.inputs import phantom

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _params(case):
    return orc.voxel_params(case.vox_struct, case.t_under, case.w_under, case.t_over, case.w_over)


# ----------------------------------------------------------------------------- O1 / O4
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_dose_and_beamlet_gradient_match_dense_product(seed):
    rng = np.random.default_rng(seed)
    n_vox, n_bl = int(rng.integers(1, 64)), int(rng.integers(1, 16))
    row_ptr, col, val, dense = phantom.random_csr(n_vox, n_bl, 0.3, seed)
    x = rng.standard_normal(n_bl)
    g = rng.standard_normal(n_vox)
    z = orc.dose(row_ptr, col, val, x)
    w = orc.beamlet_gradient(row_ptr, col, val, g, n_bl)
    D = dense.astype(np.float64)
    np.testing.assert_allclose(z, D @ x, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(w, D.T @ g, rtol=1e-13, atol=1e-14)
    # a transposed operand or an index off by one cannot pass both products and the empty row/column
    assert (np.diff(row_ptr) == 0).any() or n_vox <= 2


def test_adjoint_identity_full_size(cfg0):
    rng = np.random.default_rng(5)
    x = rng.random(cfg0.n_bl)
    g = rng.standard_normal(cfg0.n_vox)
    z = orc.dose(cfg0.row_ptr, cfg0.col_idx, cfg0.val, x)
    w = orc.beamlet_gradient(cfg0.row_ptr, cfg0.col_idx, cfg0.val, g, cfg0.n_bl)
    assert abs(w @ x - g @ z) <= 1e-11 * (abs(g) @ abs(z))


def test_beamlet_intensity_and_column_consistency(tiny):
    """eq. (7) + eq. (1),(2): D x(y) == sum_k y_k a_k for a pool of random apertures."""
    rng = np.random.default_rng(3)
    rows = 2
    beams = [0, 1, 1]
    L = np.array([[0, 1], [1, 0], [0, 2]], dtype=np.int32)
    R = np.array([[2, 3], [3, 0], [3, 3]], dtype=np.int32)
    y = rng.random(3)
    x = orc.beamlet_intensity(tiny.n_bl, beams, L, R, y, tiny.beam_row_ptr, tiny.row_bl_ptr)
    # by hand: beamlet id = (beam*rows + m)*3 + c
    x_ref = np.zeros(tiny.n_bl)
    for k, b in enumerate(beams):
        for m in range(rows):
            for c in range(L[k, m], R[k, m]):
                x_ref[(b * rows + m) * 3 + c] += y[k]
    np.testing.assert_allclose(x, x_ref, rtol=0, atol=0)
    z = orc.dose(tiny.row_ptr, tiny.col_idx, tiny.val, x)
    cols = [orc.aperture_column(tiny.row_ptr, tiny.col_idx, tiny.val,
                                orc.aperture_open_mask(tiny.n_bl, b, L[k], R[k], tiny.beam_row_ptr,
                                                       tiny.row_bl_ptr)) for k, b in enumerate(beams)]
    np.testing.assert_allclose(z, sum(yk * a for yk, a in zip(y, cols)), rtol=1e-13)
    # column against the dense matrix
    m0 = orc.aperture_open_mask(tiny.n_bl, 0, L[0], R[0], tiny.beam_row_ptr, tiny.row_bl_ptr)
    np.testing.assert_allclose(cols[0], tiny.dense @ m0.astype(np.float64), rtol=1e-13)


# ----------------------------------------------------------------------------- O2 / O3
def test_objective_at_zero_dose_closed_form(cfg0):
    """F(z = 0) = sum over targets of alpha_s (T_s^-)^2 = 10.0 for configs[0] (eq. 9)."""
    vp = _params(cfg0)
    assert orc.objective(np.zeros(cfg0.n_vox), vp) == pytest.approx(10.0, rel=1e-12)


@pytest.mark.parametrize("c", [0.0, 0.2, 0.5, 1.0, 1.02, 1.3])
def test_objective_uniform_dose_is_independent_of_structure_size(mini, c):
    vp = _params(mini)
    expect = 0.0
    for s in range(mini.n_struct):
        if not (mini.vox_struct == s).any():
            continue
        expect += float(mini.w_under[s]) * max(0.0, float(mini.t_under[s]) - c) ** 2
        expect += float(mini.w_over[s]) * max(0.0, c - float(mini.t_over[s])) ** 2
    assert orc.objective(np.full(mini.n_vox, c), vp) == pytest.approx(expect, rel=1e-11, abs=1e-15)


def test_objective_and_gradient_hand_case():
    txt = open(os.path.join(GOLDEN, "objective_hand_case.txt")).read().splitlines()
    kv = {l.split("=")[0].strip(): l.split("=")[1].strip() for l in txt if not l.startswith("#") and "=" in l}
    z = np.array([float(v) for v in kv["z"].split(",")])
    vp = orc.voxel_params(np.array([0, 0, 1, 1], dtype=np.int32), [1.0, 0.0], [10.0, 0.0], [1.05, 0.3], [5.0, 2.0])
    assert orc.objective(z, vp) == pytest.approx(float(kv["F"]), rel=1e-12)
    np.testing.assert_allclose(orc.voxel_gradient(z, vp), [float(v) for v in kv["g"].split(",")], rtol=1e-12, atol=1e-15)


def test_unlabelled_voxels_carry_no_penalty(cfg0):
    vp = _params(cfg0)
    z = np.full(cfg0.n_vox, 5.0)
    g = orc.voxel_gradient(z, vp)
    assert np.all(g[cfg0.vox_struct < 0] == 0.0)
    assert np.all(g[cfg0.vox_struct >= 0] > 0.0)


def test_voxel_gradient_central_differences(tiny):
    vp = _params(tiny)
    rng = np.random.default_rng(0)
    z = rng.uniform(0.0, 1.4, tiny.n_vox)
    # keep away from the kinks so that the piecewise quadratic is exactly differentiable nearby
    for t in (vp.tm, vp.tp):
        near = np.abs(z - t) < 1e-3
        z[near] += 5e-3
    g = orc.voxel_gradient(z, vp)
    h = 1e-5
    for j in range(tiny.n_vox):
        zp, zm = z.copy(), z.copy()
        zp[j] += h; zm[j] -= h
        fd = (orc.objective(zp, vp) - orc.objective(zm, vp)) / (2 * h)
        assert fd == pytest.approx(g[j], rel=1e-6, abs=1e-9)


def test_beamlet_gradient_is_dF_dx(tiny):
    """w_i = dF/dx_i (reading S1) by central differences on x."""
    vp = _params(tiny)
    rng = np.random.default_rng(1)
    x = rng.uniform(0.0, 0.12, tiny.n_bl)
    F = lambda xx: orc.objective(orc.dose(tiny.row_ptr, tiny.col_idx, tiny.val, xx), vp)
    z = orc.dose(tiny.row_ptr, tiny.col_idx, tiny.val, x)
    w = orc.beamlet_gradient(tiny.row_ptr, tiny.col_idx, tiny.val, orc.voxel_gradient(z, vp), tiny.n_bl)
    h = 1e-6
    for i in range(tiny.n_bl):
        xp, xm = x.copy(), x.copy()
        xp[i] += h; xm[i] -= h
        assert (F(xp) - F(xm)) / (2 * h) == pytest.approx(w[i], rel=2e-5, abs=1e-8)


# ----------------------------------------------------------------------------- O5
def _brute(w):
    """Independent O(n^2) statement: prefix sums, all 0 <= l < r <= n, ties -> smallest l then r."""
    n = len(w)
    S = np.r_[0.0, np.cumsum(w)]
    best = (0.0, 0, 0)
    for l in range(n):
        for r in range(l + 1, n + 1):
            v = S[r] - S[l]
            if v < best[0]:
                best = (v, l, r)
    return best


def test_row_pricing_golden_trace():
    for line in open(os.path.join(GOLDEN, "row_scan_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        ws, v, l, r = [p.strip() for p in line.split("|")]
        w = np.array([float(t) for t in ws.split(",")])
        for method in ("scan", "exhaustive"):
            got = orc.price_row(w, method)
            assert got == (float(v), int(l), int(r)), (method, ws, got)


def test_row_pricing_all_small_integer_rows():
    """Every row over {-2..2}^n, n <= 5: many exact ties; definition == printed scan == brute force."""
    for n in range(0, 6):
        for w in itertools.product([-2.0, -1.0, 0.0, 1.0, 2.0], repeat=n):
            w = np.array(w, dtype=np.float64)
            a = orc.price_row(w, "exhaustive")
            assert a == orc.price_row(w, "scan") == _brute(w), w


@pytest.mark.parametrize("seed", range(5))
def test_row_pricing_random_rows(seed):
    rng = np.random.default_rng(seed)
    for _ in range(300):
        n = int(rng.integers(1, 90))
        if rng.random() < 0.5:
            w = rng.standard_normal(n).astype(np.float32).astype(np.float64)
        else:
            w = rng.integers(-3, 4, n).astype(np.float64)
        a = orc.price_row(w, "exhaustive")
        b = orc.price_row(w, "scan")
        c = _brute(w)
        assert a[1:] == b[1:] == c[1:]
        assert a[0] == pytest.approx(c[0], rel=1e-13, abs=1e-13) and b[0] == pytest.approx(c[0], rel=1e-13, abs=1e-13)


def test_row_pricing_degenerate_rows():
    assert orc.price_row(np.zeros(0)) == (0.0, 0, 0)
    assert orc.price_row(np.array([3.0])) == (0.0, 0, 0)
    assert orc.price_row(np.array([-3.0])) == (-3.0, 0, 1)
    assert orc.price_row(np.zeros(7)) == (0.0, 0, 0)
    assert orc.price_row(-np.ones(9)) == (-9.0, 0, 9)


# ----------------------------------------------------------------------------- O6 / O7
def _enumerate_apertures(case, beam):
    rows = range(case.beam_row_ptr[beam], case.beam_row_ptr[beam + 1])
    per_row = []
    for r in rows:
        n = case.row_bl_ptr[r + 1] - case.row_bl_ptr[r]
        per_row.append([(0, 0)] + [(l, rr) for l in range(n) for rr in range(l + 1, n + 1)])
    for combo in itertools.product(*per_row):
        yield np.array([c[0] for c in combo], dtype=np.int32), np.array([c[1] for c in combo], dtype=np.int32)


def test_subproblem_equals_enumeration_over_all_apertures(tiny):
    """Separability: row minima summed per beam == min over all 49 apertures of a_k . pi."""
    vp = _params(tiny)
    rng = np.random.default_rng(7)
    for trial in range(5):
        z = rng.uniform(0.0, 1.5, tiny.n_vox)
        g = orc.voxel_gradient(z, vp)
        w = orc.beamlet_gradient(tiny.row_ptr, tiny.col_idx, tiny.val, g, tiny.n_bl)
        pr = orc.price(w, tiny.beam_row_ptr, tiny.row_bl_ptr)
        best = []
        for b in range(tiny.n_beams):
            vals = []
            for le, ri in _enumerate_apertures(tiny, b):
                m = orc.aperture_open_mask(tiny.n_bl, b, le, ri, tiny.beam_row_ptr, tiny.row_bl_ptr)
                a = tiny.dense @ m.astype(np.float64)          # column straight from the dense matrix
                vals.append(float(a @ g))
            assert len(vals) == 49
            best.append(min(vals))
            assert pr.beam_price[b] == pytest.approx(min(vals), rel=1e-10, abs=1e-12)
        assert pr.best_beam == int(np.argmin(best))
        assert pr.price == pytest.approx(min(best), rel=1e-10, abs=1e-12)


def test_first_iteration_closed_form(mini):
    """With an empty pool z = 0: pi_j = -2 alpha_s T_s^- / |v_s| on targets, 0 elsewhere, so every
    w_i <= 0, every row opens from its first column to its last column with w < 0, and the beam is
    argmax_b sum_{i in b} sum_{j in targets} (alpha_s T_s^- / |v_s|) D_ji."""
    vp = _params(mini)
    g = orc.voxel_gradient(np.zeros(mini.n_vox), vp)
    tgt = mini.w_under[np.clip(mini.vox_struct, 0, None)] > 0
    tgt &= mini.vox_struct >= 0
    assert np.all(g[~tgt] == 0.0) and np.all(g[tgt] < 0.0)
    w = orc.beamlet_gradient(mini.row_ptr, mini.col_idx, mini.val, g, mini.n_bl)
    assert np.all(w <= 0.0)
    pr = orc.price(w, mini.beam_row_ptr, mini.row_bl_ptr)
    per_beam = [w[mini.row_bl_ptr[mini.beam_row_ptr[b]]: mini.row_bl_ptr[mini.beam_row_ptr[b + 1]]].sum()
                for b in range(mini.n_beams)]
    assert pr.best_beam == int(np.argmin(per_beam))
    for r in range(mini.n_rows):
        wr = w[mini.row_bl_ptr[r]: mini.row_bl_ptr[r + 1]]
        neg = np.nonzero(wr < 0)[0]
        if neg.size == 0:
            assert (pr.left[r], pr.right[r]) == (0, 0)
        else:
            assert (pr.left[r], pr.right[r]) == (0, neg[-1] + 1)
