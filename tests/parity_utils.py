"""Helpers of the GPU parity tests: the north star's comparison rules written once.

Nothing here is used by the product path.  The "second best interval" table is a numpy
restatement of the plain definition (all intervals of a row), independent of both the oracle's C
code and the CUDA kernel.
"""
import numpy as np

from oracle import dao_oracle as orc


def interval_table(w):
    """All interval sums of one row: T[l, r] = w[l] + .. + w[r-1] for 0 <= l < r <= n (fp64), inf elsewhere."""
    w = np.asarray(w, dtype=np.float64)
    n = w.size
    S = np.r_[0.0, np.cumsum(w)]
    T = S[None, :] - S[:, None]
    T[np.tril_indices(n + 1)] = np.inf
    return T


def row_gap(w, left, right):
    """Smallest value among the candidates other than the chosen one minus the chosen value.
    Candidates = the closed row (value 0, counted once) + every non-empty interval."""
    T = interval_table(w)
    chosen = 0.0 if left == right else T[left, right]
    if left != right:
        T = T.copy()
        T[left, right] = np.inf
        others = min(float(T.min()), 0.0)
    else:
        others = float(T.min())           # closed row chosen: best non-empty interval
    return others - chosen, chosen


def check_rows(w32, row_bl_ptr, left, right, vstar, rel_gap=1e-6):
    """North-star rule: with the same fp32 w, leaf positions are bit-exact whenever best and
    second-best intervals differ by more than rel_gap * max(|v*|, max|w_i|); rows inside the band
    must still reach v* to rel_gap.  Returns (#rows compared exactly, #rows inside the band)."""
    w = np.asarray(w32, dtype=np.float32).astype(np.float64)
    pr_exact = pr_band = 0
    for r in range(len(row_bl_ptr) - 1):
        seg = w[row_bl_ptr[r]:row_bl_ptr[r + 1]]
        v_o, l_o, r_o = orc.price_row(seg, "exhaustive")
        scale = max(abs(v_o), float(np.max(np.abs(seg))) if seg.size else 0.0, 1e-300)
        gap, _ = row_gap(seg, l_o, r_o)
        assert abs(vstar[r] - v_o) <= rel_gap * scale, (r, vstar[r], v_o)
        if gap > rel_gap * scale:
            assert (int(left[r]), int(right[r])) == (l_o, r_o), (r, left[r], right[r], l_o, r_o, gap)
            pr_exact += 1
        else:
            # any interval reaching v* within the band is acceptable; it must be a valid interval
            n = seg.size
            assert 0 <= left[r] <= right[r] <= n
            got = float(seg[left[r]:right[r]].sum())
            assert abs(got - v_o) <= rel_gap * scale
            pr_band += 1
    return pr_exact, pr_band


def check_beam(beam_price_gpu, best_gpu, beam_price_orc, rel_gap=1e-6):
    bp = np.asarray(beam_price_orc, dtype=np.float64)
    order = np.argsort(bp, kind="stable")
    scale = max(float(np.max(np.abs(bp))), 1e-300)
    np.testing.assert_allclose(beam_price_gpu, bp, rtol=0, atol=1e-9 * scale)
    if bp.size == 1 or bp[order[1]] - bp[order[0]] > rel_gap * scale:
        assert int(best_gpu) == int(order[0])
    else:
        assert abs(bp[int(best_gpu)] - bp[order[0]]) <= rel_gap * scale


def oracle_state_from_plan(ph, beams, lefts, rights, y):
    """z, g, w of the oracle at the intensities (y over the given apertures)."""
    vp = orc.voxel_params_of(ph)
    K = len(beams)
    max_rows = int(np.max(np.diff(ph.beam_row_ptr)))
    L = np.zeros((K, max_rows), np.int32); R = np.zeros_like(L)
    for k in range(K):
        L[k, :len(lefts[k])] = lefts[k]; R[k, :len(rights[k])] = rights[k]
    x = orc.beamlet_intensity(ph.n_bl, np.asarray(beams, np.int32), L, R, np.asarray(y, np.float64),
                              ph.beam_row_ptr, ph.row_bl_ptr) if K else np.zeros(ph.n_bl)
    z = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x)
    g = orc.voxel_gradient(z, vp)
    w = orc.beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, g, ph.n_bl)
    return vp, x, z, g, w, orc.objective(z, vp)


def oracle_columns(ph, beams, lefts, rights):
    A = np.zeros((len(beams), ph.n_vox))
    for k, b in enumerate(beams):
        A[k] = orc.aperture_column(ph.row_ptr, ph.col_idx, ph.val,
                                   orc.aperture_open_mask(ph.n_bl, b, lefts[k], rights[k], ph.beam_row_ptr, ph.row_bl_ptr))
    return A
