"""Pins of the oracle's re-optimisation mode (PAPER.md:254 with eq. 3-5):
alpha_j = beta_j = 1, T_j = a reference dose, under-dose penalised on target voxels only."""
import os

import numpy as np

from oracle import dao_oracle as orc
from paper_1003_5402_b200.inputs import phantom

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "reopt_hand_case.txt")


class FourVoxels:
    vox_struct = np.array([0, 1, 0, 1], np.int32)
    t_under = np.zeros(2, np.float32); t_over = np.zeros(2, np.float32)
    w_under = np.array([1.0, 0.0], np.float32); w_over = np.array([1.0, 1.0], np.float32)
    per_voxel_weights = True


def test_hand_case_from_the_definition():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    tgt = np.array([int(r[1]) for r in rows]); T = np.array([float(r[2]) for r in rows])
    z = np.array([float(r[3]) for r in rows])
    f_expect = sum(float(r[4]) + float(r[5]) for r in rows)
    g_expect = np.array([float(r[6]) for r in rows])
    case = FourVoxels()
    case.vox_struct = np.where(tgt == 1, 0, 1).astype(np.int32)
    case.vox_threshold = T.astype(np.float32)
    vp = orc.voxel_params_of(case)
    T32 = T.astype(np.float32).astype(np.float64)      # thresholds are stored in fp32
    np.testing.assert_array_equal(vp.tm, T32); np.testing.assert_array_equal(vp.tp, T32)
    np.testing.assert_array_equal(vp.a, tgt.astype(float)); np.testing.assert_array_equal(vp.b, np.ones(4))
    assert abs(orc.objective(z, vp) - f_expect) < 1e-7 and abs(f_expect - 0.09) < 1e-15
    np.testing.assert_allclose(orc.voxel_gradient(z, vp), g_expect, atol=1e-6)


def test_closed_forms_on_a_phantom(mini_reopt):
    ph = mini_reopt
    vp = orc.voxel_params_of(ph)
    T = ph.vox_threshold.astype(np.float64)
    n_t = int((ph.vox_struct == 0).sum())
    assert n_t > 0 and ph.n_struct == 2 and ph.per_voxel_weights
    assert orc.objective(T, vp) == 0.0                                   # reproducing the reference costs nothing
    c = 0.125
    assert abs(orc.objective(T + c, vp) - ph.n_vox * c * c) < 1e-9       # over-dose on every voxel, beta = 1
    assert abs(orc.objective(T - c, vp) - n_t * c * c) < 1e-9            # under-dose on targets only, alpha = 1
    g = orc.voxel_gradient(T + c, vp)
    np.testing.assert_allclose(g, 2 * c, atol=1e-12)
    g = orc.voxel_gradient(T - c, vp)
    np.testing.assert_allclose(g, np.where(ph.vox_struct == 0, -2 * c, 0.0), atol=1e-12)


def test_gradient_by_finite_differences(mini_reopt):
    ph = mini_reopt
    vp = orc.voxel_params_of(ph)
    rng = np.random.default_rng(3)
    z = ph.vox_threshold.astype(np.float64) + rng.normal(0, 0.2, ph.n_vox)
    g = orc.voxel_gradient(z, vp)
    for j in rng.integers(0, ph.n_vox, 40):
        h = 1e-6
        zp, zm = z.copy(), z.copy(); zp[j] += h; zm[j] -= h
        fd = (orc.objective(zp, vp) - orc.objective(zm, vp)) / (2 * h)
        assert abs(fd - g[j]) <= 1e-5 * max(1.0, abs(g[j]))


def test_plan_objective_decreases_and_terminal_prices(mini_reopt):
    plan = orc.run(mini_reopt, 8)
    f = [plan.history[0].objective_before] + [h.objective for h in plan.history]
    assert all(b <= a * (1 + 1e-12) for a, b in zip(f, f[1:])) and f[-1] < 0.8 * f[0]
    assert all(h.price < 0 for h in plan.history)
    # F(0) closed form: sum of T_j^2 over target voxels
    T = mini_reopt.vox_threshold.astype(np.float64)
    assert abs(f[0] - float((T[mini_reopt.vox_struct == 0] ** 2).sum())) < 1e-9 * f[0]


def test_recipe_is_seeded_and_shaped_like_a_dose(mini_reopt):
    again = phantom.make("mini_reopt", seed=0)
    np.testing.assert_array_equal(again.vox_threshold, mini_reopt.vox_threshold)
    other = phantom.make("mini_reopt", seed=1)
    assert other.n_vox != mini_reopt.n_vox or not np.array_equal(other.vox_threshold, mini_reopt.vox_threshold)
    T = mini_reopt.vox_threshold
    assert T.dtype == np.float32 and np.isfinite(T).all() and T.min() > 0 and T.max() < 1.1 * mini_reopt.prescription
    assert T[mini_reopt.vox_struct == 0].mean() > 2 * T[mini_reopt.vox_struct == 1].mean()
