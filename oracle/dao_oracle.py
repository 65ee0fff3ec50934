"""ctypes front end of the fp64 CPU oracle (``dao_oracle.c``) plus the column-generation driver.

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module.  It imports
nothing from the CUDA package, and the CUDA package imports nothing from here.

The driver :func:`run` is O9 of DESIGN.md: the column-generation loop of PAPER.md:114, 134, 169
(Figure 1): price -> add the best aperture -> re-solve the restricted master problem, until
``max_apertures`` apertures or until the sub-problem finds no improving aperture.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dao_oracle.c")
_LIB = os.path.join(_HERE, "libdao_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, no OpenMP).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_objective.restype = C.c_double
        _lib.orc_master_gradient.restype = C.c_double
        _lib.orc_master_pg.restype = C.c_int32
        _lib.orc_master_newton.restype = C.c_int32
        _lib.orc_fmo_pg.restype = C.c_int32
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


# ----------------------------------------------------------------------------- steps
def dose(row_ptr, col_idx, val, x):
    """O1: z = D x (eq. 1 with eq. 2, 7)."""
    row_ptr, col_idx, val, x = _i32(row_ptr), _i32(col_idx), _f32(val), _f64(x)
    n_vox = row_ptr.size - 1
    z = np.empty(n_vox, dtype=np.float64)
    lib().orc_dose(C.c_int32(n_vox), _p(row_ptr), _p(col_idx), _p(val), _p(x), _p(z))
    return z


@dataclass
class VoxelParams:
    a: np.ndarray
    b: np.ndarray
    tm: np.ndarray
    tp: np.ndarray


def voxel_params(vox_struct, t_under, w_under, t_over, w_over) -> VoxelParams:
    """Per-voxel alpha_s/|v_s|, beta_s/|v_s|, T_s^-, T_s^+ of eq. (9)-(10)."""
    vs = _i32(vox_struct)
    n = vs.size
    tu, wu, to, wo = _f64(t_under), _f64(w_under), _f64(t_over), _f64(w_over)
    out = [np.empty(n, dtype=np.float64) for _ in range(4)]
    lib().orc_voxel_params(C.c_int32(n), _p(vs), C.c_int32(tu.size), _p(tu), _p(wu), _p(to), _p(wo),
                           *[_p(o) for o in out])
    return VoxelParams(*out)


def voxel_params_of(ph) -> VoxelParams:
    """Per-voxel penalty parameters of a problem instance.  Default: eq. (9)-(10).  With
    ``ph.per_voxel_weights`` the weights are the alpha_j, beta_j of eq. (3)-(4) as given (no division
    by |v_s|); with ``ph.vox_threshold`` T_j replaces both thresholds -- together the paper's
    re-optimisation mode (alpha_j = beta_j = 1, T_j = reference dose)."""
    vp = voxel_params(ph.vox_struct, ph.t_under, ph.w_under, ph.t_over, ph.w_over)
    vs = _i32(ph.vox_struct)
    inside = vs >= 0
    if getattr(ph, "per_voxel_weights", False):
        a = np.zeros(vs.size); b = np.zeros(vs.size)
        a[inside] = _f64(ph.w_under)[vs[inside]]
        b[inside] = _f64(ph.w_over)[vs[inside]]
        vp = VoxelParams(a, b, vp.tm, vp.tp)
    vt = getattr(ph, "vox_threshold", None)
    if vt is not None:
        t = np.asarray(vt, dtype=np.float32).astype(np.float64)
        vp = VoxelParams(vp.a, vp.b, t.copy(), t.copy())
    return vp


def objective(z, vp: VoxelParams) -> float:
    """O2: F(z), eq. (3)-(5) / (9)-(10)."""
    z = _f64(z)
    return float(lib().orc_objective(C.c_int32(z.size), _p(z), _p(vp.a), _p(vp.b), _p(vp.tm), _p(vp.tp)))


def voxel_gradient(z, vp: VoxelParams):
    """O3: pi_j = dF/dz_j."""
    z = _f64(z)
    g = np.empty_like(z)
    lib().orc_voxel_gradient(C.c_int32(z.size), _p(z), _p(vp.a), _p(vp.b), _p(vp.tm), _p(vp.tp), _p(g))
    return g


def beamlet_gradient(row_ptr, col_idx, val, g, n_bl):
    """O4: w_i = sum_j D_ij pi_j."""
    row_ptr, col_idx, val, g = _i32(row_ptr), _i32(col_idx), _f32(val), _f64(g)
    w = np.empty(n_bl, dtype=np.float64)
    lib().orc_beamlet_gradient(C.c_int32(row_ptr.size - 1), C.c_int32(n_bl), _p(row_ptr), _p(col_idx),
                               _p(val), _p(g), _p(w))
    return w


def price_row(w, method: str = "exhaustive"):
    """O5: one leaf row -> (v*, left, right), half-open.  method: 'exhaustive' (plain definition)
    or 'scan' (the paper's printed scan)."""
    w = _f64(w)
    v = C.c_double(0.0); l = C.c_int32(0); r = C.c_int32(0)
    fn = lib().orc_price_row_exhaustive if method == "exhaustive" else lib().orc_price_row_scan
    fn(C.c_int32(w.size), _p(w), C.byref(v), C.byref(l), C.byref(r))
    return v.value, l.value, r.value


@dataclass
class Pricing:
    vstar: np.ndarray
    left: np.ndarray
    right: np.ndarray
    beam_price: np.ndarray
    best_beam: int

    @property
    def price(self) -> float:
        return float(self.beam_price[self.best_beam])


def price(w, beam_row_ptr, row_bl_ptr) -> Pricing:
    """O5 + O6: the sub-problem (8)."""
    w, brp, rbp = _f64(w), _i32(beam_row_ptr), _i32(row_bl_ptr)
    n_beams, n_rows = brp.size - 1, rbp.size - 1
    vs = np.zeros(n_rows, dtype=np.float64)
    le = np.zeros(n_rows, dtype=np.int32)
    ri = np.zeros(n_rows, dtype=np.int32)
    bp = np.zeros(n_beams, dtype=np.float64)
    bb = C.c_int32(-1)
    lib().orc_price(_p(w), C.c_int32(n_beams), _p(brp), _p(rbp), _p(vs), _p(le), _p(ri), _p(bp), C.byref(bb))
    return Pricing(vs, le, ri, bp, bb.value)


def price_jaws(w, beam_row_ptr, row_bl_ptr, row_col0=None) -> Pricing:
    """Jaws-only sub-problem (reading J1): the best RECTANGLE per beam (consecutive rows, one
    common lateral range), all rectangles enumerated.  row_col0[r] = lateral position of row r's first beamlet."""
    w, brp, rbp = _f64(w), _i32(beam_row_ptr), _i32(row_bl_ptr)
    n_beams, n_rows = brp.size - 1, rbp.size - 1
    rc0 = _i32(np.zeros(n_rows) if row_col0 is None else row_col0)
    vs = np.zeros(n_rows, dtype=np.float64)
    le = np.zeros(n_rows, dtype=np.int32)
    ri = np.zeros(n_rows, dtype=np.int32)
    bp = np.zeros(n_beams, dtype=np.float64)
    bb = C.c_int32(-1)
    lib().orc_price_jaws(_p(w), C.c_int32(n_beams), _p(brp), _p(rbp), _p(rc0), _p(vs), _p(le), _p(ri), _p(bp), C.byref(bb))
    return Pricing(vs, le, ri, bp, bb.value)


MLC_MODES = {"consecutive": 0, "jaws": 1, "interdigitation": 2, "connected": 3}


def price_chain(w, beam_row_ptr, row_bl_ptr, row_col0=None, mlc: str = "interdigitation") -> Pricing:
    """Sub-problem under the interdigitation (reading J2) or connectedness (reading J3) constraint
    (PAPER.md:260): dynamic programme over the leaf rows of every beam.  Only the value is unique."""
    w, brp, rbp = _f64(w), _i32(beam_row_ptr), _i32(row_bl_ptr)
    n_beams, n_rows = brp.size - 1, rbp.size - 1
    rc0 = _i32(np.zeros(n_rows) if row_col0 is None else row_col0)
    vs = np.zeros(n_rows, dtype=np.float64)
    le = np.zeros(n_rows, dtype=np.int32)
    ri = np.zeros(n_rows, dtype=np.int32)
    bp = np.zeros(n_beams, dtype=np.float64)
    bb = C.c_int32(-1)
    lib().orc_price_chain(C.c_int32(MLC_MODES[mlc]), _p(w), C.c_int32(n_beams), _p(brp), _p(rbp), _p(rc0), _p(vs),
                          _p(le), _p(ri), _p(bp), C.byref(bb))
    return Pricing(vs, le, ri, bp, bb.value)


def aperture_open_mask(n_bl, beam, left, right, beam_row_ptr, row_bl_ptr):
    """0/1 mask over beamlets of an aperture in `beam` with per-row half-open leaves (rows of that beam)."""
    m = np.zeros(n_bl, dtype=np.uint8)
    for k, r in enumerate(range(beam_row_ptr[beam], beam_row_ptr[beam + 1])):
        m[row_bl_ptr[r] + left[k]: row_bl_ptr[r] + right[k]] = 1
    return m


def aperture_column(row_ptr, col_idx, val, open_mask):
    """O7: a_j = sum_{i in A} D_ij (eq. 2)."""
    row_ptr, col_idx, val = _i32(row_ptr), _i32(col_idx), _f32(val)
    om = np.ascontiguousarray(open_mask, dtype=np.uint8)
    a = np.empty(row_ptr.size - 1, dtype=np.float64)
    lib().orc_aperture_column(C.c_int32(row_ptr.size - 1), _p(row_ptr), _p(col_idx), _p(val), _p(om), _p(a))
    return a


def beamlet_intensity(n_bl, ap_beam, ap_left, ap_right, y, beam_row_ptr, row_bl_ptr):
    """eq. (7): x_i = sum_{k in K_i} y_k.  ap_left/right: [n_ap, max_rows] int32."""
    ap_beam = _i32(ap_beam); y = _f64(y)
    ap_left = _i32(ap_left).reshape(len(ap_beam), -1)
    ap_right = _i32(ap_right).reshape(len(ap_beam), -1)
    x = np.zeros(n_bl, dtype=np.float64)
    lib().orc_beamlet_intensity(C.c_int32(n_bl), C.c_int32(len(ap_beam)), _p(ap_beam), _p(ap_left),
                                _p(ap_right), C.c_int32(ap_left.shape[1] if len(ap_beam) else 0), _p(y),
                                _p(_i32(beam_row_ptr)), _p(_i32(row_bl_ptr)), _p(x))
    return x


@dataclass
class MasterResult:
    y: np.ndarray
    objective: float
    n_iter: int
    kkt: float


def master(A, y0, vp: VoxelParams, tol: float = 1e-10, max_iter: int = 20000,
           method: str = "newton") -> MasterResult:
    """O8: min_{y>=0} F(A y).  A: [K, n_vox] float64 aperture-major.  method 'pg' = gradient
    projection with exact line search (the method the paper names), 'newton' = projected Newton."""
    A = _f64(A)
    K, n_vox = A.shape
    y = _f64(y0).copy()
    f = C.c_double(0.0); kkt = C.c_double(0.0)
    fn = lib().orc_master_pg if method == "pg" else lib().orc_master_newton
    it = fn(C.c_int32(n_vox), C.c_int32(K), _p(A), _p(y), _p(vp.a), _p(vp.b), _p(vp.tm), _p(vp.tp),
            C.c_double(tol), C.c_int32(max_iter), C.byref(f), C.byref(kkt))
    return MasterResult(y, f.value, int(it), kkt.value)


def master_gradient(A, y, vp: VoxelParams):
    """(F(A y), dF/dy) -- for KKT checks."""
    A = _f64(A); y = _f64(y)
    K, n_vox = A.shape
    grad = np.zeros(K, dtype=np.float64)
    f = lib().orc_master_gradient(C.c_int32(n_vox), C.c_int32(K), _p(A), _p(y), _p(vp.a), _p(vp.b),
                                  _p(vp.tm), _p(vp.tp), _p(grad))
    return float(f), grad


def dense_transpose(ph) -> np.ndarray:
    """D^T as a dense [n_bl, n_vox] fp64 array (small instances only): the "aperture" block whose
    columns are the single beamlets, i.e. the FMO model in the master's notation."""
    A = np.zeros((ph.n_bl, ph.n_vox), dtype=np.float64)
    rp = _i32(ph.row_ptr)
    rows = np.repeat(np.arange(ph.n_vox), np.diff(rp))
    A[_i32(ph.col_idx), rows] = _f32(ph.val).astype(np.float64)
    return A


def fmo(ph, x0=None, tol: float = 1e-10, max_iter: int = 20000, method: str = "newton") -> MasterResult:
    """FMO: min_{x >= 0} F(D x) over the beamlet intensities.
    method 'pg' = plain gradient projection on the sparse D (orc_fmo_pg, any size); 'newton' = the
    master's projected Newton on the dense D^T (small instances; same optimum value by convexity)."""
    vp = voxel_params_of(ph)
    x = np.zeros(ph.n_bl) if x0 is None else _f64(x0).copy()
    if method == "newton":
        return master(dense_transpose(ph), x, vp, tol, max_iter, "newton")
    rp, ci, v = _i32(ph.row_ptr), _i32(ph.col_idx), _f32(ph.val)
    f = C.c_double(0.0); kkt = C.c_double(0.0)
    it = lib().orc_fmo_pg(C.c_int32(ph.n_vox), C.c_int32(ph.n_bl), _p(rp), _p(ci), _p(v), _p(x), _p(vp.a), _p(vp.b),
                          _p(vp.tm), _p(vp.tp), C.c_double(tol), C.c_int32(max_iter), C.byref(f), C.byref(kkt))
    return MasterResult(x, f.value, int(it), kkt.value)


# ----------------------------------------------------------------------------- driver (O9)
@dataclass
class Iteration:
    k: int                     # pool size after this iteration
    beam: int
    price: float               # reduced cost of the aperture added
    left: np.ndarray           # leaves of the rows of `beam`
    right: np.ndarray
    objective_before: float    # F at the master optimum of the previous pool (F(0) for the first)
    objective: float           # F at the master optimum including the new aperture
    n_master_iter: int
    kkt: float


@dataclass
class Plan:
    beams: List[int] = field(default_factory=list)
    lefts: List[np.ndarray] = field(default_factory=list)
    rights: List[np.ndarray] = field(default_factory=list)
    y: np.ndarray = field(default_factory=lambda: np.zeros(0))
    objective: float = float("nan")
    converged: bool = False
    stalled: bool = False          # stopped on a duplicate candidate after an unconverged master (reading S6)
    n_duplicates: int = 0
    history: List[Iteration] = field(default_factory=list)
    A: Optional[np.ndarray] = None


def price_converged(pr: Pricing, w, beam_row_ptr, price_tol: float) -> bool:
    """Reading S3: optimal iff price_b* >= -price_tol * max_i |w_i| * (rows in b*)."""
    rows = int(beam_row_ptr[pr.best_beam + 1] - beam_row_ptr[pr.best_beam])
    return pr.price >= -price_tol * float(np.max(np.abs(w))) * rows


def run(ph, max_apertures: int, master_tol: float = 1e-10, master_max_iter: int = 20000,
        price_tol: float = 1e-9, method: str = "newton", keep_A: bool = False, mlc: str = "consecutive",
        stop_on_duplicate: bool = True) -> Plan:
    """O9: the column-generation loop.  `ph` is any object with the Phantom fields.  mlc = "consecutive"
    (the paper's experiments) or "jaws" (jaws-only delivery, reading J1).

    stop_on_duplicate (reading S6; the paper is silent): a candidate that equals an aperture k of the
    pool has the reduced cost dF/dy_k of the master, >= 0 at the master's optimum, so its negative price is residue
    of the master solve and, being the minimum over all apertures, bounds every other reduced cost.  The loop then
    stops: `converged` if that master solve met its stopping test and the residue is of the size the solve reports
    (-price <= 10 max(kkt, price tolerance)), `stalled` otherwise (appending the same column again cannot help).
    With the default tolerances (1e-10) the rule never fires; False appends the duplicate (SURVEY's first reading)."""
    vp = voxel_params_of(ph)
    n_vox, n_bl = ph.n_vox, ph.n_bl
    A = np.zeros((max_apertures, n_vox), dtype=np.float64)
    plan = Plan()
    y = np.zeros(0, dtype=np.float64)
    z = np.zeros(n_vox, dtype=np.float64)
    f_cur = objective(z, vp)
    for it in range(max_apertures):
        g = voxel_gradient(z, vp)
        w = beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, g, n_bl)
        if mlc == "jaws":
            pr = price_jaws(w, ph.beam_row_ptr, ph.row_bl_ptr, getattr(ph, "row_col0", None))
        elif mlc in ("interdigitation", "connected"):
            pr = price_chain(w, ph.beam_row_ptr, ph.row_bl_ptr, getattr(ph, "row_col0", None), mlc)
        else:
            pr = price(w, ph.beam_row_ptr, ph.row_bl_ptr)
        if price_converged(pr, w, ph.beam_row_ptr, price_tol):
            plan.converged = True
            break
        b = pr.best_beam
        r0, r1 = int(ph.beam_row_ptr[b]), int(ph.beam_row_ptr[b + 1])
        le, ri = pr.left[r0:r1].copy(), pr.right[r0:r1].copy()
        if stop_on_duplicate and any(pb == b and np.array_equal(pl, le) and np.array_equal(prr, ri)
                                     for pb, pl, prr in zip(plan.beams, plan.lefts, plan.rights)):
            plan.n_duplicates += 1
            last = plan.history[-1]
            tol_abs = price_tol * float(np.max(np.abs(w))) * (r1 - r0)
            if last.n_master_iter < master_max_iter and -pr.price <= 10.0 * max(last.kkt, tol_abs):
                plan.converged = True
            else:
                plan.stalled = True
            break
        A[it] = aperture_column(ph.row_ptr, ph.col_idx, ph.val,
                                aperture_open_mask(n_bl, b, le, ri, ph.beam_row_ptr, ph.row_bl_ptr))
        y = np.r_[y, 0.0]
        res = master(A[:it + 1], y, vp, master_tol, master_max_iter, method)
        y = res.y
        plan.beams.append(b); plan.lefts.append(le); plan.rights.append(ri)
        plan.history.append(Iteration(it + 1, b, pr.price, le, ri, f_cur, res.objective, res.n_iter, res.kkt))
        f_cur = res.objective
        # dose of the current plan through the beamlet matrix (eq. 1, 2, 7)
        max_rows = int(np.max(np.diff(ph.beam_row_ptr)))
        L = np.zeros((it + 1, max_rows), dtype=np.int32); R = np.zeros_like(L)
        for k in range(it + 1):
            L[k, :plan.lefts[k].size] = plan.lefts[k]; R[k, :plan.rights[k].size] = plan.rights[k]
        x = beamlet_intensity(n_bl, plan.beams, L, R, y, ph.beam_row_ptr, ph.row_bl_ptr)
        z = dose(ph.row_ptr, ph.col_idx, ph.val, x)
    plan.y = y
    plan.objective = objective(z, vp)
    if keep_A:
        plan.A = A[:len(plan.beams)].copy()
    return plan
