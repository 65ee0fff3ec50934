"""``dao_price_from_w_static``: the pricing step for callers that cannot allocate.

Every other call of the library runs inside a context whose workspace came from ``cudaMalloc``.  A host
process whose device memory was handed out in full at start-up, a plug-in that receives device pointers but
no allocator, or a delivery-time loop whose rules forbid ``cudaMalloc`` / ``cudaFree`` (both synchronise the
device and can fail late) has no way to get one.  For them the library carries its intermediate arrays in a
fixed 136 KiB array of its own image and takes only the caller's inputs and outputs.

What is checked here: on the same device vectors the new entry point returns exactly what the existing
context path (``dao_price_from_w``) returns -- the two run the same row kernel body and the same tail, so
leaves, best beam, row minima and beam prices must agree bit for bit, which is the bar the pricing parity
tests use -- and it does so on two calls in a row, the second on a smaller, different problem, so that
anything the first call left in the shared array (ticket, max|w| entries beyond the second problem's rows)
would show.  The file sorts last on purpose: ``pytest -x`` stops at the first failure and this test must
not hide the parity suite.  It passes alone in a fresh process (first use of the array on the device) and
after the other tests.
"""
import ctypes as C

import numpy as np
import pytest


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_sizes_beyond_the_fixed_array_are_refused():
    """No GPU needed: the limits are checked before any CUDA call, with the limit named in the message."""
    from paper_1003_5402_b200 import build, dao
    build.build()
    lib = dao.load_library()
    p = C.c_void_p(256)            # never dereferenced: the call must fail on the sizes alone
    for n_rows, n_beams in ((dao.STATIC_MAX_ROWS + 1, 4), (100, dao.STATIC_MAX_BEAMS + 1)):
        st = lib.dao_price_from_w_static(p, p, p, C.c_int32(n_rows), C.c_int32(n_beams), p, p, p, p, p, None)
        assert st == 2, st                                                      # DAO_E_SHAPE
        msg = lib.dao_last_error(None).decode()
        assert "DAO_STATIC_MAX_ROWS = 16384" in msg and "DAO_STATIC_MAX_BEAMS = 1024" in msg, msg
    assert lib.dao_price_from_w_static(p, p, p, C.c_int32(0), C.c_int32(1), p, p, p, p, p, None) == 1   # DAO_E_ARG
    assert lib.dao_price_from_w_static(None, p, p, C.c_int32(4), C.c_int32(1), p, p, p, p, p, None) == 1
    assert b"null" in lib.dao_last_error(None)


@pytest.mark.gpu
def test_static_pricing_matches_the_context_path_twice(mini):
    import torch
    from paper_1003_5402_b200 import dao
    from paper_1003_5402_b200.inputs import phantom

    # first call: 3000 rows of 80 beamlets in 75 beams; second call: 257 rows of 33 in 7 beams
    # (fewer rows, fewer beams, rows that span two 32-wide tiles with a ragged tail)
    cases = [phantom.pricing_rows(3000, 80, rows_per_beam=40, seed=11),
             phantom.pricing_rows(257, 33, rows_per_beam=40, seed=12)]
    # integer-valued rows: exact sums, many exact ties -- exercises the fixed tie-break as well
    rng = np.random.default_rng(13)
    rows = [rng.integers(-2, 3, n).astype(np.float32) for n in rng.integers(1, 70, 300)]
    rbp = np.r_[0, np.cumsum([r.size for r in rows])].astype(np.int32)
    cases.append((np.concatenate(rows), np.array([0, 100, 100, 250, 300], np.int32), rbp))   # one beam without rows

    got, want = [], []
    # the static entry point first, back to back, no context alive, nothing synchronised in between
    for w, brp, rbp in cases:
        got.append(dao.price_from_w_static(_dev(w), _dev(rbp), _dev(brp)))
    torch.cuda.synchronize()
    got = [[t.cpu().numpy() for t in g] for g in got]
    # the existing path
    with dao.Dao(mini) as d:
        for w, brp, rbp in cases:
            want.append([t.cpu().numpy() for t in d.price_from_w(_dev(w), _dev(rbp), _dev(brp))])
        # and once more with a context alive and its kernels in between (shared array must not care)
        w, brp, rbp = cases[1]
        d.price()
        again = [t.cpu().numpy() for t in dao.price_from_w_static(_dev(w), _dev(rbp), _dev(brp))]
    for g, e in zip(got + [again], want + [want[1]]):
        for name, a, b in zip(("left", "right", "vstar", "beam_price", "best"), g, e):
            assert a.dtype == b.dtype and a.shape == b.shape, name
            assert np.array_equal(a, b), f"{name} differs from dao_price_from_w"
    # caller-held outputs are written in place (the C call allocates nothing; neither need the wrapper)
    w, brp, rbp = cases[0]
    out = (torch.full((3000,), -7, dtype=torch.int32, device="cuda"), torch.full((3000,), -7, dtype=torch.int32, device="cuda"),
           torch.full((3000,), 9.0, dtype=torch.float64, device="cuda"), torch.full((75,), 9.0, dtype=torch.float64, device="cuda"),
           torch.full((1,), -7, dtype=torch.int32, device="cuda"))
    wd, rd, bd = _dev(w), _dev(rbp), _dev(brp)
    free_before = torch.cuda.mem_get_info()[0]
    ret = dao.price_from_w_static(wd, rd, bd, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # the device's free memory did not move
    assert all(r.data_ptr() == o.data_ptr() for r, o in zip(ret, out))
    for a, b in zip(out, want[0]):
        assert np.array_equal(a.cpu().numpy(), b)
