"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every function
include/dao.h declares; the ctypes structs mirror the header; without a CUDA device the product
path fails loudly instead of falling back; the product never imports the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dao.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1003_5402_b200 import build, dao
    build.build()
    return dao.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dao_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_function_is_exported(lib):
    from paper_1003_5402_b200 import dao
    names = _declared_functions()
    assert {"dao_create", "dao_price", "dao_solve_master", "dao_run", "dao_get_plan"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in dao.h but not exported"
    assert sorted(dao.EXPORTS) == names


def test_default_options_and_struct_layout(lib):
    from paper_1003_5402_b200 import dao
    o = dao.default_options()
    assert (o.k_max, o.master_max_iter, o.master_method, o.timers) == (50, 2000, 2, 1)
    assert o.master_tol == 1e-7 and o.price_tol == 1e-6 and o.master_ls_tol == 0.01
    # sizes the C side was compiled with (natural alignment, no packing)
    assert C.sizeof(dao.COptions) == 56 and C.sizeof(dao.CMlc) == 32 and C.sizeof(dao.CStructs) == 72 and C.sizeof(dao.CCsr) == 48 and C.sizeof(dao.CPriceInfo) == 48
    assert C.sizeof(dao.CMasterInfo) == 48 and C.sizeof(dao.CIterRecord) == 56 == dao.ITER_RECORD_DTYPE.itemsize
    assert C.sizeof(dao.CRunInfo) == 112 and C.sizeof(dao.CPlan) == 64 and C.sizeof(dao.CDims) == 56


def test_argument_errors_need_no_gpu(lib):
    from paper_1003_5402_b200 import dao
    sizes = dao.CSizes()
    assert lib.dao_workspace_bytes(None, None, None, None, C.byref(sizes)) == 1          # DAO_E_ARG
    assert b"null" in lib.dao_last_error(None)
    rp = np.array([0, 1], np.int32); ci = np.array([0], np.int32); v = np.array([1.0], np.float32)
    vs = np.array([0], np.int32); t = np.array([1.0], np.float32)
    csr = dao.CCsr(1, 1, 1, rp.ctypes.data, ci.ctypes.data, v.ctypes.data, 0)
    mlc = dao.CMlc(1, 1, rp.ctypes.data, rp.ctypes.data)
    st = dao.CStructs(1, vs.ctypes.data, t.ctypes.data, t.ctypes.data, t.ctypes.data, t.ctypes.data)
    opt = dao.default_options(k_max=dao.MAX_APERTURES + 1)
    assert lib.dao_workspace_bytes(C.byref(csr), C.byref(mlc), C.byref(st), C.byref(opt), C.byref(sizes)) == 6
    bad_mlc = dao.CMlc(1, 1, rp.ctypes.data, np.array([0, 2], np.int32).ctypes.data)
    opt = dao.default_options()
    assert lib.dao_workspace_bytes(C.byref(csr), C.byref(bad_mlc), C.byref(st), C.byref(opt), C.byref(sizes)) == 2
    assert lib.dao_get_dims(None, None) == 1 and lib.dao_destroy(None) == 0


def test_no_cpu_fallback(lib, tiny):
    """Without a CUDA device the product path raises; it never computes on the CPU."""
    import torch
    from paper_1003_5402_b200 import dao
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(RuntimeError, match="CUDA"):
        dao.Dao(tiny)
    rp = np.ascontiguousarray(tiny.row_ptr); ci = np.ascontiguousarray(tiny.col_idx); v = np.ascontiguousarray(tiny.val)
    vs = np.ascontiguousarray(tiny.vox_struct)
    csr = dao.CCsr(tiny.n_vox, tiny.n_bl, tiny.nnz, rp.ctypes.data, ci.ctypes.data, v.ctypes.data, 0)
    mlc = dao.CMlc(tiny.n_beams, tiny.n_rows, tiny.beam_row_ptr.ctypes.data, tiny.row_bl_ptr.ctypes.data)
    st = dao.CStructs(2, vs.ctypes.data, tiny.t_under.ctypes.data, tiny.w_under.ctypes.data,
                      tiny.t_over.ctypes.data, tiny.w_over.ctypes.data)
    sizes = dao.CSizes()
    opt = dao.default_options()
    assert lib.dao_workspace_bytes(C.byref(csr), C.byref(mlc), C.byref(st), C.byref(opt), C.byref(sizes)) == 3   # DAO_E_CUDA
    assert b"CUDA" in lib.dao_last_error(None)


def test_product_and_oracle_share_nothing():
    """Neither side imports, includes or reads the other (the input generator serves both)."""
    pkg = os.path.join(ROOT, "paper_1003_5402_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                code = "\n".join(l for l in text.splitlines() if not l.strip().startswith(("//", "#", "*", "/*")))
                assert "import oracle" not in code and "from oracle" not in code and "dao_oracle" not in code, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1003_5402_b200" not in text and "from paper_1003_5402_b200" not in text, f
            assert "dao.h" not in text and "libdao.so" not in text, f
