"""Thin ctypes binding of ``include/dao.h`` (argument marshalling only).

PyTorch is used for exactly two things here: allocating the device buffers the C library works
in (``torch.empty(..., device="cuda")``) and naming the CUDA stream.  Every step of the hot path
runs in the kernels of ``libdao.so``; there is no CPU fallback -- if the library or a CUDA device
is missing, construction fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdao.so")

DAO_OK = 0
STATUS_NAMES = {0: "DAO_OK", 1: "DAO_E_ARG", 2: "DAO_E_SHAPE", 3: "DAO_E_CUDA", 4: "DAO_E_ALLOC",
                5: "DAO_E_STATE", 6: "DAO_E_UNSUPPORTED"}
MEM_HOST, MEM_DEVICE = 0, 1
MLC_CONSECUTIVE, MLC_JAWS_ONLY, MLC_INTERDIGITATION, MLC_CONNECTED = 0, 1, 2, 3
MAX_APERTURES = 128
(VEC_Z, VEC_G, VEC_W, VEC_X, VEC_Y, VEC_VSTAR, VEC_LEFT, VEC_RIGHT, VEC_BEAM_PRICE, VEC_HISTORY,
 VEC_MASTER_Z, VEC_MASTER_PHASES, VEC_ITER_SECONDS) = range(13)

EXPORTS = ["dao_default_options", "dao_workspace_bytes", "dao_create", "dao_price", "dao_solve_master",
           "dao_run", "dao_get_plan", "dao_reset", "dao_destroy", "dao_last_error", "dao_get_vector",
           "dao_get_dims", "dao_spmv", "dao_spmv_t", "dao_eval_x", "dao_price_from_w", "dao_set_pool",
           "dao_resolve_master", "dao_fmo_solve", "dao_price_from_w_static"]
STATIC_MAX_ROWS, STATIC_MAX_BEAMS = 16384, 1024     # DAO_STATIC_MAX_ROWS / DAO_STATIC_MAX_BEAMS of dao.h


class DaoError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


# ----------------------------------------------------------------------------- C structs
class CCsr(C.Structure):
    _fields_ = [("n_vox", C.c_int32), ("n_bl", C.c_int32), ("nnz", C.c_int64), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p), ("mem", C.c_int)]


class CMlc(C.Structure):
    _fields_ = [("n_beams", C.c_int32), ("n_rows", C.c_int32), ("beam_row_ptr", C.c_void_p),
                ("row_bl_ptr", C.c_void_p), ("row_col0", C.c_void_p)]


class CStructs(C.Structure):
    _fields_ = [("n_struct", C.c_int32), ("vox_struct", C.c_void_p), ("t_under", C.c_void_p),
                ("w_under", C.c_void_p), ("t_over", C.c_void_p), ("w_over", C.c_void_p),
                ("vox_threshold", C.c_void_p), ("per_voxel_weights", C.c_int32), ("struct_count", C.c_void_p)]


class COptions(C.Structure):
    _fields_ = [("k_max", C.c_int32), ("master_max_iter", C.c_int32), ("master_tol", C.c_double),
                ("price_tol", C.c_double), ("master_ls_tol", C.c_double), ("master_method", C.c_int32), ("sell_sigma", C.c_int32),
                ("timers", C.c_int32), ("mlc_mode", C.c_int32), ("reserved", C.c_int32), ("pad_", C.c_int32)]


class CSizes(C.Structure):
    _fields_ = [("workspace_bytes", C.c_size_t), ("scratch_bytes", C.c_size_t)]


class CPriceInfo(C.Structure):
    _fields_ = [("beam", C.c_int32), ("converged", C.c_int32), ("price", C.c_double), ("objective", C.c_double),
                ("w_abs_max", C.c_double), ("n_open_beamlets", C.c_int32), ("duplicate", C.c_int32),
                ("stalled", C.c_int32), ("reserved", C.c_int32)]


class CMasterInfo(C.Structure):
    _fields_ = [("n_apertures", C.c_int32), ("n_pg_iter", C.c_int32), ("hit_max_iter", C.c_int32),
                ("n_restarts", C.c_int32), ("objective", C.c_double), ("kkt_residual", C.c_double),
                ("pg_norm", C.c_double), ("n_passes", C.c_int32), ("reserved", C.c_int32)]


class CRunInfo(C.Structure):
    _fields_ = [("n_apertures", C.c_int32), ("n_iterations", C.c_int32), ("converged", C.c_int32),
                ("n_duplicates", C.c_int32), ("n_pg_iter_total", C.c_int64), ("objective", C.c_double),
                ("seconds_total", C.c_double), ("seconds_intensity", C.c_double), ("seconds_spmv", C.c_double),
                ("seconds_spmv_t", C.c_double), ("seconds_price", C.c_double), ("seconds_column", C.c_double),
                ("seconds_master", C.c_double), ("n_passes_total", C.c_int64), ("n_hit_max_iter", C.c_int32),
                ("n_kernel_launches", C.c_int32), ("stalled", C.c_int32), ("reserved", C.c_int32)]


class CIterRecord(C.Structure):
    _fields_ = [("k", C.c_int32), ("beam", C.c_int32), ("n_pg_iter", C.c_int32), ("duplicate", C.c_int32),
                ("price", C.c_double), ("objective_before", C.c_double), ("objective", C.c_double),
                ("kkt_residual", C.c_double), ("n_passes", C.c_int32), ("hit_max_iter", C.c_int32)]


class CFmoInfo(C.Structure):
    _fields_ = [("n_iter", C.c_int32), ("converged", C.c_int32), ("hit_max_iter", C.c_int32), ("n_restarts", C.c_int32),
                ("n_ls_evals", C.c_int32), ("reserved", C.c_int32), ("objective", C.c_double),
                ("kkt_residual", C.c_double), ("pg_norm", C.c_double), ("seconds", C.c_double)]


class CPlan(C.Structure):
    _fields_ = [("cap_apertures", C.c_int32), ("cap_rows", C.c_int32), ("n_apertures", C.c_int32),
                ("n_rows_used", C.c_int32), ("beam", C.c_void_p), ("intensity", C.c_void_p),
                ("ap_row_ptr", C.c_void_p), ("left", C.c_void_p), ("right", C.c_void_p), ("objective", C.c_double)]


class CDims(C.Structure):
    _fields_ = [("n_vox", C.c_int32), ("n_bl", C.c_int32), ("n_beams", C.c_int32), ("n_rows", C.c_int32),
                ("n_struct", C.c_int32), ("k_max", C.c_int32), ("nnz", C.c_int64), ("sell_elems", C.c_int64),
                ("sell_slice_rows", C.c_int32), ("sell_sigma", C.c_int32), ("n_sm", C.c_int32), ("master_method", C.c_int32)]


ITER_RECORD_DTYPE = np.dtype([("k", "<i4"), ("beam", "<i4"), ("n_pg_iter", "<i4"), ("duplicate", "<i4"),
                              ("price", "<f8"), ("objective_before", "<f8"), ("objective", "<f8"),
                              ("kkt_residual", "<f8"), ("n_passes", "<i4"), ("hit_max_iter", "<i4")])

_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libdao.so (building is the job of :mod:`paper_1003_5402_b200.build`)."""
    global _lib
    if _lib is None or path is not None:
        p = path or LIB_PATH
        if not os.path.exists(p):
            raise FileNotFoundError(f"{p} not found: run `python -m paper_1003_5402_b200.build` "
                                    "(there is no CPU fallback)")
        lib = C.CDLL(p)
        lib.dao_last_error.restype = C.c_char_p
        lib.dao_last_error.argtypes = [C.c_void_p]
        for name in EXPORTS:
            fn = getattr(lib, name)
            if name not in ("dao_last_error", "dao_default_options"):
                fn.restype = C.c_int
        lib.dao_default_options.restype = None
        _lib = lib
    return _lib


def default_options(**overrides) -> COptions:
    o = COptions()
    load_library().dao_default_options(C.byref(o))
    for k, v in overrides.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown option {k}")
        setattr(o, k, v)
    return o


def _np_ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def price_from_w_static(w_dev, row_bl_ptr_dev, beam_row_ptr_dev, out=None, stream=None):
    """``dao_price_from_w_static``: steps 5-6 (row pricing, beam sums, best beam) on device tensors with no
    :class:`Dao` context and no device allocation inside the library -- for hosts that own ``w`` and the MLC
    tables but may not (or cannot) call ``cudaMalloc`` when they need the answer; the library's intermediate
    arrays live in a fixed 136 KiB array of ``libdao.so`` instead of a workspace.  At most ``STATIC_MAX_ROWS``
    leaf rows and ``STATIC_MAX_BEAMS`` beams (``DaoError`` with ``DAO_E_SHAPE`` beyond).  All calls on a GPU
    share that array: keep them on one stream or order them, overlapping calls race.  The first call on a
    device looks the array's address up; make it at start-up.

    ``out`` = ``(left, right, vstar, beam_price, best)`` device tensors (int32 [n_rows] x 2, float64 [n_rows],
    float64 [n_beams], int32 [1]) the caller already holds; when None this wrapper creates them with torch --
    a convenience of the Python side only, the C call itself takes them as arguments.  ``stream``: a
    ``torch.cuda.Stream`` (default: torch's current stream).  Asynchronous; returns the five tensors."""
    import torch
    lib = load_library()
    n_rows, n_beams = row_bl_ptr_dev.numel() - 1, beam_row_ptr_dev.numel() - 1
    for t, dt in ((w_dev, torch.float32), (row_bl_ptr_dev, torch.int32), (beam_row_ptr_dev, torch.int32)):
        assert t.is_cuda and t.dtype == dt and t.is_contiguous()
    if out is None:
        out = (torch.empty(max(n_rows, 0), dtype=torch.int32, device=w_dev.device),
               torch.empty(max(n_rows, 0), dtype=torch.int32, device=w_dev.device),
               torch.empty(max(n_rows, 0), dtype=torch.float64, device=w_dev.device),
               torch.empty(max(n_beams, 0), dtype=torch.float64, device=w_dev.device),
               torch.empty(1, dtype=torch.int32, device=w_dev.device))
    le, ri, vs, bp, best = out
    for t, dt, n in ((le, torch.int32, n_rows), (ri, torch.int32, n_rows), (vs, torch.float64, n_rows),
                     (bp, torch.float64, n_beams), (best, torch.int32, 1)):
        assert t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() >= n
    s = torch.cuda.current_stream(w_dev.device) if stream is None else stream
    with torch.cuda.device(w_dev.device):
        st = lib.dao_price_from_w_static(C.c_void_p(w_dev.data_ptr()), C.c_void_p(row_bl_ptr_dev.data_ptr()),
                                         C.c_void_p(beam_row_ptr_dev.data_ptr()), C.c_int32(n_rows), C.c_int32(n_beams),
                                         C.c_void_p(le.data_ptr()), C.c_void_p(ri.data_ptr()), C.c_void_p(vs.data_ptr()),
                                         C.c_void_p(bp.data_ptr()), C.c_void_p(best.data_ptr()), C.c_void_p(s.cuda_stream))
    if st != DAO_OK:
        raise DaoError(st, (lib.dao_last_error(None) or b"").decode())
    return le, ri, vs, bp, best


@dataclass
class Plan:
    beams: np.ndarray          # int32 [K]
    intensity: np.ndarray      # float32 [K]
    ap_row_ptr: np.ndarray     # int32 [K+1]
    left: np.ndarray           # int32 [rows used]
    right: np.ndarray
    objective: float

    def leaves(self, k: int):
        s, e = self.ap_row_ptr[k], self.ap_row_ptr[k + 1]
        return self.left[s:e], self.right[s:e]


class Dao:
    """One DAO context.  ``ph`` is any object with the fields of
    :class:`paper_1003_5402_b200.inputs.phantom.Phantom` (numpy arrays = host inputs); pass
    ``device_inputs=True`` to upload the CSR with torch first and hand device pointers over."""

    def __init__(self, ph, device_inputs: bool = False, stream=None, **options):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1003_5402_b200.dao needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.lib = load_library()
        self.opt = default_options(**options)
        self.n_vox, self.n_bl, self.nnz = int(ph.n_vox), int(ph.n_bl), int(ph.nnz)
        self.n_beams, self.n_rows = int(ph.n_beams), int(ph.n_rows)
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        self._keep: List[object] = []

        row_ptr = np.ascontiguousarray(ph.row_ptr, dtype=np.int32)
        col_idx = np.ascontiguousarray(ph.col_idx, dtype=np.int32)
        val = np.ascontiguousarray(ph.val, dtype=np.float32)
        vs = np.ascontiguousarray(ph.vox_struct, dtype=np.int32)
        brp = np.ascontiguousarray(ph.beam_row_ptr, dtype=np.int32)
        rbp = np.ascontiguousarray(ph.row_bl_ptr, dtype=np.int32)
        tu = np.ascontiguousarray(ph.t_under, dtype=np.float32)
        wu = np.ascontiguousarray(ph.w_under, dtype=np.float32)
        to = np.ascontiguousarray(ph.t_over, dtype=np.float32)
        wo = np.ascontiguousarray(ph.w_over, dtype=np.float32)
        self._keep += [row_ptr, col_idx, val, vs, brp, rbp, tu, wu, to, wo]
        csr = CCsr(self.n_vox, self.n_bl, self.nnz)
        st = CStructs(int(tu.size))
        if device_inputs:
            d_rp, d_ci, d_v, d_vs = (torch.from_numpy(a).cuda() for a in (row_ptr, col_idx, val, vs))
            self._keep += [d_rp, d_ci, d_v, d_vs]
            csr.row_ptr, csr.col_idx, csr.val, csr.mem = d_rp.data_ptr(), d_ci.data_ptr(), d_v.data_ptr(), MEM_DEVICE
            st.vox_struct = d_vs.data_ptr()
        else:
            csr.row_ptr, csr.col_idx, csr.val, csr.mem = _np_ptr(row_ptr), _np_ptr(col_idx), _np_ptr(val), MEM_HOST
            st.vox_struct = _np_ptr(vs)
        st.t_under, st.w_under, st.t_over, st.w_over = _np_ptr(tu), _np_ptr(wu), _np_ptr(to), _np_ptr(wo)
        # re-optimisation mode: per-voxel thresholds T_j, weights not divided by |v_s|
        vt = getattr(ph, "vox_threshold", None)
        st.per_voxel_weights = 1 if getattr(ph, "per_voxel_weights", False) else 0
        if vt is not None:
            vt = np.ascontiguousarray(vt, dtype=np.float32)
            if vt.size != self.n_vox:
                raise ValueError("vox_threshold must have n_vox entries")
            if device_inputs:
                d_vt = torch.from_numpy(vt).cuda()
                self._keep.append(d_vt)
                st.vox_threshold = d_vt.data_ptr()
            else:
                self._keep.append(vt)
                st.vox_threshold = _np_ptr(vt)
        # voxel-row slab: |v_s| of the whole problem, see paper_1003_5402_b200.sharded
        sc = getattr(ph, "struct_count", None)
        if sc is not None:
            sc = np.ascontiguousarray(sc, dtype=np.int64)
            if sc.size != tu.size:
                raise ValueError("struct_count must have n_struct entries")
            self._keep.append(sc)
            st.struct_count = _np_ptr(sc)
        mlc = CMlc(self.n_beams, self.n_rows, _np_ptr(brp), _np_ptr(rbp))
        rc0 = getattr(ph, "row_col0", None)
        if rc0 is not None:
            rc0 = np.ascontiguousarray(rc0, dtype=np.int32)
            if rc0.size != self.n_rows:
                raise ValueError("row_col0 must have n_rows entries")
            self._keep.append(rc0)
            mlc.row_col0 = _np_ptr(rc0)

        sizes = CSizes()
        rc = self.lib.dao_workspace_bytes(C.byref(csr), C.byref(mlc), C.byref(st), C.byref(self.opt), C.byref(sizes))
        if rc != DAO_OK:
            raise DaoError(rc, self.lib.dao_last_error(None).decode())
        self.workspace_bytes, self.scratch_bytes = int(sizes.workspace_bytes), int(sizes.scratch_bytes)
        with torch.cuda.stream(self._stream):
            self._workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device="cuda")
            scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device="cuda")
        self._ctx = C.c_void_p()
        rc = self.lib.dao_create(C.byref(csr), C.byref(mlc), C.byref(st), C.byref(self.opt),
                                 C.c_void_p(self._workspace.data_ptr()), C.c_size_t(self.workspace_bytes),
                                 C.c_void_p(scratch.data_ptr()), C.c_size_t(self.scratch_bytes),
                                 C.c_void_p(self._stream.cuda_stream), C.byref(self._ctx))
        del scratch
        if rc != DAO_OK:
            self._ctx = C.c_void_p()
            raise DaoError(rc, self.lib.dao_last_error(None).decode())
        if device_inputs:          # inputs are only read during dao_create
            self._keep = self._keep[:10]

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc: int):
        if rc != DAO_OK:
            raise DaoError(rc, self.lib.dao_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.dao_destroy(self._ctx)
            self._ctx = C.c_void_p()
        self._workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ------------------------------------------------------------------ the five entry points
    def price(self) -> CPriceInfo:
        info = CPriceInfo()
        self._check(self.lib.dao_price(self._ctx, C.byref(info)))
        return info

    def solve_master(self) -> CMasterInfo:
        info = CMasterInfo()
        self._check(self.lib.dao_solve_master(self._ctx, C.byref(info)))
        return info

    def resolve_master(self) -> CMasterInfo:
        info = CMasterInfo()
        self._check(self.lib.dao_resolve_master(self._ctx, C.byref(info)))
        return info

    def run(self, max_apertures: int) -> CRunInfo:
        info = CRunInfo()
        self._check(self.lib.dao_run(self._ctx, C.c_int32(max_apertures), C.byref(info)))
        return info

    def fmo_solve(self, max_iter: int = 2000, tol: float = 0.0, warm_start: bool = False) -> CFmoInfo:
        """FMO workload: min_{x >= 0} F(D x) by projected gradient on the device."""
        info = CFmoInfo()
        self._check(self.lib.dao_fmo_solve(self._ctx, C.c_int32(max_iter), C.c_double(tol),
                                           C.c_int32(1 if warm_start else 0), C.byref(info)))
        return info

    def get_plan(self) -> Plan:
        k_max = int(self.opt.k_max)
        max_rows = int(np.max(np.diff(self._keep[4]))) if self.n_beams else 0
        beam = np.zeros(k_max, np.int32); inten = np.zeros(k_max, np.float32)
        arp = np.zeros(k_max + 1, np.int32)
        le = np.zeros(max(1, k_max * max_rows), np.int32); ri = np.zeros_like(le)
        p = CPlan(k_max, int(le.size), 0, 0, _np_ptr(beam), _np_ptr(inten), _np_ptr(arp), _np_ptr(le), _np_ptr(ri), 0.0)
        self._check(self.lib.dao_get_plan(self._ctx, C.byref(p)))
        K, R = int(p.n_apertures), int(p.n_rows_used)
        return Plan(beam[:K].copy(), inten[:K].copy(), arp[:K + 1].copy(), le[:R].copy(), ri[:R].copy(), float(p.objective))

    def reset(self):
        self._check(self.lib.dao_reset(self._ctx))

    # ------------------------------------------------------------------ hooks
    def dims(self) -> CDims:
        d = CDims()
        self._check(self.lib.dao_get_dims(self._ctx, C.byref(d)))
        return d

    def get_vector(self, which: int) -> np.ndarray:
        k_max = int(self.opt.k_max)
        shapes = {VEC_Z: (self.n_vox, np.float32), VEC_G: (self.n_vox, np.float32), VEC_W: (self.n_bl, np.float32),
                  VEC_X: (self.n_bl, np.float32), VEC_Y: (k_max, np.float64), VEC_VSTAR: (self.n_rows, np.float64),
                  VEC_LEFT: (self.n_rows, np.int32), VEC_RIGHT: (self.n_rows, np.int32),
                  VEC_BEAM_PRICE: (self.n_beams, np.float64), VEC_HISTORY: (k_max, ITER_RECORD_DTYPE),
                  VEC_MASTER_Z: (self.n_vox, np.float64), VEC_MASTER_PHASES: (16, np.uint64),
                  VEC_ITER_SECONDS: (k_max * 6, np.float64)}
        n, dt = shapes[which]
        out = np.zeros(n, dtype=dt)
        self._check(self.lib.dao_get_vector(self._ctx, C.c_int32(which), C.c_void_p(_np_ptr(out)), C.c_int(MEM_HOST)))
        return out

    def spmv(self, x_dev, z_dev=None):
        """z = D x on device tensors (float32); asynchronous on the context's stream."""
        torch = self._torch
        if z_dev is None:
            z_dev = torch.empty(self.n_vox, dtype=torch.float32, device="cuda")
        assert x_dev.is_cuda and x_dev.dtype == torch.float32 and x_dev.numel() == self.n_bl and x_dev.is_contiguous()
        self._check(self.lib.dao_spmv(self._ctx, C.c_void_p(x_dev.data_ptr()), C.c_void_p(z_dev.data_ptr())))
        return z_dev

    def spmv_t(self, g_dev, w_dev=None):
        """w = D^T g on device tensors (float32); asynchronous on the context's stream."""
        torch = self._torch
        if w_dev is None:
            w_dev = torch.empty(self.n_bl, dtype=torch.float32, device="cuda")
        assert g_dev.is_cuda and g_dev.dtype == torch.float32 and g_dev.numel() == self.n_vox and g_dev.is_contiguous()
        self._check(self.lib.dao_spmv_t(self._ctx, C.c_void_p(g_dev.data_ptr()), C.c_void_p(w_dev.data_ptr())))
        return w_dev

    def eval_x(self, x_dev) -> float:
        f = C.c_double(0.0)
        assert x_dev.is_cuda and x_dev.numel() == self.n_bl and x_dev.is_contiguous()
        self._check(self.lib.dao_eval_x(self._ctx, C.c_void_p(x_dev.data_ptr()), C.byref(f)))
        return f.value

    def price_from_w(self, w_dev, row_bl_ptr_dev=None, beam_row_ptr_dev=None):
        """Steps 5-6 on a device fp32 vector.  Returns device tensors (left, right, vstar, beam_price, best)."""
        torch = self._torch
        if row_bl_ptr_dev is None:
            n_rows, n_beams, rp, bp = self.n_rows, self.n_beams, None, None
        else:
            n_rows, n_beams = row_bl_ptr_dev.numel() - 1, beam_row_ptr_dev.numel() - 1
            rp, bp = C.c_void_p(row_bl_ptr_dev.data_ptr()), C.c_void_p(beam_row_ptr_dev.data_ptr())
        le = torch.empty(n_rows, dtype=torch.int32, device="cuda"); ri = torch.empty_like(le)
        vs = torch.empty(n_rows, dtype=torch.float64, device="cuda")
        bpz = torch.empty(n_beams, dtype=torch.float64, device="cuda")
        best = torch.empty(1, dtype=torch.int32, device="cuda")
        self._check(self.lib.dao_price_from_w(self._ctx, C.c_void_p(w_dev.data_ptr()), rp, bp,
                                              C.c_int32(0 if rp is None else n_rows), C.c_int32(0 if rp is None else n_beams),
                                              C.c_void_p(le.data_ptr()), C.c_void_p(ri.data_ptr()), C.c_void_p(vs.data_ptr()),
                                              C.c_void_p(bpz.data_ptr()), C.c_void_p(best.data_ptr())))
        return le, ri, vs, bpz, best

    def set_pool(self, beams, lefts, rights, y=None):
        """Replace the pool: beams[k], lefts[k]/rights[k] = leaves of the rows of that beam."""
        K = len(beams)
        beam = np.ascontiguousarray(beams, dtype=np.int32)
        arp = np.zeros(K + 1, np.int32)
        for k in range(K):
            arp[k + 1] = arp[k] + len(lefts[k])
        le = np.ascontiguousarray(np.concatenate([np.asarray(a, np.int32) for a in lefts]) if K else np.zeros(0, np.int32))
        ri = np.ascontiguousarray(np.concatenate([np.asarray(a, np.int32) for a in rights]) if K else np.zeros(0, np.int32))
        yy = None if y is None else np.ascontiguousarray(y, dtype=np.float64)
        self._check(self.lib.dao_set_pool(self._ctx, C.c_int32(K), C.c_void_p(_np_ptr(beam)), C.c_void_p(_np_ptr(arp)),
                                          C.c_void_p(_np_ptr(le)), C.c_void_p(_np_ptr(ri)),
                                          None if yy is None else C.c_void_p(_np_ptr(yy))))
