"""Seeded synthetic IMRT phantoms: the INPUT generator shared by the oracle and the CUDA path.

This module produces inputs only -- the sparse beamlet dose-deposition matrix D (CSR, fp32
values, int32 indices), the MLC leaf-row tables and the structure / prescription tables of
BASELINE.json's configs.  It holds none of the method's arithmetic (no dose product, no
objective, no gradient, no pricing, no master solve); neither ``oracle/`` nor the CUDA library
is imported here, and both consume the arrays it returns byte for byte.

The phantoms stand in for the paper's ten clinical cases (Table 1), which are
not available.  The recipe follows BASELINE.json configs[0..4]:

* voxel centres on a regular grid centred at the isocentre, x fastest, then y, then z;
* body = elliptical cylinder along z; structures = spheres / ellipsoids / z-cylinders, one
  structure per voxel by priority (targets by descending prescription, then OARs in listed
  order, then body);
* coplanar parallel beams: gantry angle t travels along d = (sin t, -cos t, 0) (gantry 0 goes
  along -y); leaves travel along u = (cos t, sin t, 0); leaf rows stack along z;
* D[v, j] = exp(-0.005/mm * depth_v) * exp(-r_vj^2 / (2 * (4 mm)^2)), depth_v = path length from
  the point where the voxel's ray enters the body ellipse, r_vj = lateral distance between the
  voxel centre and beamlet j's central ray; entries below 1e-3 of the column maximum dropped;
* beamlets are numbered beam-major, then leaf row, then left to right; each leaf row is the
  contiguous hull of the beamlets kept in it, so a row is a contiguous slice of beamlet ids;
* a seeded sub-voxel offset on every structure centre and a seeded offset on the first gantry
  angle break the exact mirror symmetry of the prostate geometry (exact beam ties otherwise).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

MU_PER_MM = 0.005      # attenuation, BASELINE.json configs[0]
SIGMA_MM = 4.0         # lateral Gaussian sigma, BASELINE.json configs[0]
REL_CUTOFF = 1e-3      # entries below this fraction of the column maximum are dropped
# lateral search window: exp(-r^2/32) >= 1e-3 * colmax/att_v with colmax/att_v >= ~0.13
# (0.9 * exp(-0.005*400)) gives r <= 16.9 mm; 17.5 mm leaves margin.
WINDOW_MM = 17.5


# --------------------------------------------------------------------------- shapes
@dataclass
class Shape:
    """kind: 'ellipsoid' (centre c, semi-axes r) or 'zcyl' (centre c, radius r[0], half-length r[2])."""
    kind: str
    c: Tuple[float, float, float]
    r: Tuple[float, float, float]

    def contains(self, x, y, z, shift=(0.0, 0.0, 0.0)):
        cx, cy, cz = (self.c[0] + shift[0], self.c[1] + shift[1], self.c[2] + shift[2])
        if self.kind == "ellipsoid":
            return ((x - cx) / self.r[0]) ** 2 + ((y - cy) / self.r[1]) ** 2 + ((z - cz) / self.r[2]) ** 2 <= 1.0
        if self.kind == "zcyl":
            return (((x - cx) ** 2 + (y - cy) ** 2) <= self.r[0] ** 2) & (np.abs(z - cz) <= self.r[2])
        raise ValueError(self.kind)


@dataclass
class StructureSpec:
    name: str
    shapes: List[Shape]            # union
    t_under: float                 # T_s^-   (eq. 9)
    w_under: float                 # alpha_s (0 for non-targets)
    t_over: float                  # T_s^+   (eq. 10)
    w_over: float                  # beta_s
    is_target: bool = False


@dataclass
class PhantomSpec:
    name: str
    grid: Tuple[int, int, int]                 # nx, ny, nz
    voxel_mm: float
    body_axes_mm: Tuple[float, float]          # semi-axes of the body ellipse (x, y)
    structures: List[StructureSpec]            # priority order (first wins)
    body: Optional[StructureSpec]              # penalty on remaining in-body voxels, or None (-1)
    n_beams: int
    beamlet_mm: Tuple[float, float]            # (along leaf travel u, along z)
    field: str                                 # 'fixed' (fixed_grid) or 'ptv' (pruned to PTV projection)
    fixed_grid: Tuple[int, int] = (0, 0)       # (columns, rows) when field == 'fixed'
    ptv_margin_mm: float = 5.0
    gantry_start_deg: float = 0.0
    jitter: bool = True                        # seeded symmetry breaking (reading P6)


@dataclass
class Phantom:
    name: str
    seed: int
    n_vox: int
    n_bl: int
    nnz: int
    row_ptr: np.ndarray        # int32 [n_vox+1]
    col_idx: np.ndarray        # int32 [nnz], ascending within a row
    val: np.ndarray            # float32 [nnz]
    n_beams: int
    n_rows: int
    beam_row_ptr: np.ndarray   # int32 [n_beams+1]
    row_bl_ptr: np.ndarray     # int32 [n_rows+1]
    n_struct: int
    vox_struct: np.ndarray     # int32 [n_vox], -1 = no penalty
    t_under: np.ndarray        # float32 [n_struct]
    w_under: np.ndarray
    t_over: np.ndarray
    w_over: np.ndarray
    struct_names: List[str] = field(default_factory=list)
    gantry_deg: List[float] = field(default_factory=list)
    vox_grid_index: Optional[np.ndarray] = None   # int64 [n_vox] linear index into the grid
    grid: Tuple[int, int, int] = (0, 0, 0)
    voxel_mm: float = 0.0
    prescription: float = 1.0                     # the largest target prescription
    # re-optimisation mode: per-voxel threshold T_j replacing T_s^- and T_s^+, and
    # weights used as they are (eq. 3-4) instead of divided by |v_s| (eq. 9-10)
    vox_threshold: Optional[np.ndarray] = None    # float32 [n_vox] or None
    per_voxel_weights: bool = False
    # lateral position (in beamlet widths, relative to the beam's leftmost beamlet) of the first beamlet of
    # every leaf row: rows are contiguous hulls that need not start at the same place.  Needed by the MLC
    # constraints that couple neighbouring rows (jaws-only delivery)
    row_col0: Optional[np.ndarray] = None         # int32 [n_rows] or None (= all zero)

    def summary(self) -> Dict[str, object]:
        rows = np.diff(self.row_bl_ptr)
        return {"name": self.name, "seed": self.seed, "n_vox": self.n_vox, "n_bl": self.n_bl,
                "nnz": self.nnz, "n_beams": self.n_beams, "n_rows": self.n_rows,
                "max_row_len": int(rows.max()) if rows.size else 0,
                "nnz_per_vox": self.nnz / max(1, self.n_vox), "nnz_per_bl": self.nnz / max(1, self.n_bl)}


# --------------------------------------------------------------------------- generation
def _in_body_voxels(spec: PhantomSpec):
    nx, ny, nz = spec.grid
    h = spec.voxel_mm
    xs = (np.arange(nx) - (nx - 1) / 2.0) * h
    ys = (np.arange(ny) - (ny - 1) / 2.0) * h
    zs = (np.arange(nz) - (nz - 1) / 2.0) * h
    ax, ay = spec.body_axes_mm
    inside2d = (xs[None, :] / ax) ** 2 + (ys[:, None] / ay) ** 2 <= 1.0     # [ny, nx]
    iy, ix = np.nonzero(inside2d)                                            # row-major: y then x
    n2 = ix.size
    # x fastest, then y, then z
    lin2 = iy.astype(np.int64) * nx + ix
    lin = (np.arange(nz, dtype=np.int64)[:, None] * (nx * ny) + lin2[None, :]).ravel()
    x = np.tile(xs[ix], nz)
    y = np.tile(ys[iy], nz)
    z = np.repeat(zs, n2)
    return lin, x, y, z


def _assign_structures(spec: PhantomSpec, x, y, z, rng):
    n = x.size
    sid = np.full(n, -1, dtype=np.int32)
    h = spec.voxel_mm
    names, tu, wu, to, wo = [], [], [], [], []
    for s_idx, st in enumerate(spec.structures):
        shift = tuple(rng.uniform(-h / 2, h / 2, size=3)) if spec.jitter else (0.0, 0.0, 0.0)
        m = np.zeros(n, dtype=bool)
        for sh in st.shapes:
            m |= sh.contains(x, y, z, shift)
        sid[(sid < 0) & m] = s_idx
        names.append(st.name); tu.append(st.t_under); wu.append(st.w_under)
        to.append(st.t_over); wo.append(st.w_over)
    if spec.body is not None:
        sid[sid < 0] = len(names)
        b = spec.body
        names.append(b.name); tu.append(b.t_under); wu.append(b.w_under)
        to.append(b.t_over); wo.append(b.w_over)
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    return sid, names, f32(tu), f32(wu), f32(to), f32(wo)


def _beam_cells(spec: PhantomSpec, u, zc, target_mask):
    """Beamlet cell grid for one beam.  Returns (cell_to_bl [ncz, ncu] local ids or -1,
    row lengths list, u0, z0) with cell centres at u0 + i*bu, z0 + m*bz."""
    bu, bz = spec.beamlet_mm
    if spec.field == "fixed":
        ncu, ncz = spec.fixed_grid
        u0 = -(ncu - 1) / 2.0 * bu
        z0 = -(ncz - 1) / 2.0 * bz
        keep = np.ones((ncz, ncu), dtype=bool)
    else:
        ut, zt = u[target_mask], zc[target_mask]
        m = spec.ptv_margin_mm
        # cell centres on a lattice symmetric about the isocentre: (i + 0.5) * pitch
        iu_lo = int(np.floor((ut.min() - m) / bu - 0.5)) - 1
        iu_hi = int(np.ceil((ut.max() + m) / bu - 0.5)) + 1
        iz_lo = int(np.floor((zt.min() - m) / bz - 0.5)) - 1
        iz_hi = int(np.ceil((zt.max() + m) / bz - 0.5)) + 1
        ncu, ncz = iu_hi - iu_lo + 1, iz_hi - iz_lo + 1
        u0, z0 = (iu_lo + 0.5) * bu, (iz_lo + 0.5) * bz
        keep = np.zeros((ncz, ncu), dtype=bool)
        # a beamlet is kept when its central ray passes within `m` of a projected target voxel
        cu = np.rint((ut - u0) / bu).astype(np.int64)
        cz = np.rint((zt - z0) / bz).astype(np.int64)
        ru, rz = int(np.ceil(m / bu)) + 1, int(np.ceil(m / bz)) + 1
        for dz in range(-rz, rz + 1):
            for du in range(-ru, ru + 1):
                iu, iz = cu + du, cz + dz
                ok = (iu >= 0) & (iu < ncu) & (iz >= 0) & (iz < ncz)
                d2 = (u0 + iu * bu - ut) ** 2 + (z0 + iz * bz - zt) ** 2
                ok &= d2 <= m * m
                keep[iz[ok], iu[ok]] = True
    cell_to_bl = np.full((ncz, ncu), -1, dtype=np.int64)
    row_len = []
    row_lo = []                                       # lateral cell index of each row's first beamlet
    row_z = []
    nb = 0
    for m_ in range(ncz):
        cols = np.nonzero(keep[m_])[0]
        if cols.size == 0:
            continue
        lo, hi = int(cols[0]), int(cols[-1])          # contiguous hull of the row (reading S7)
        n = hi - lo + 1
        cell_to_bl[m_, lo:hi + 1] = nb + np.arange(n)
        row_len.append(n)
        row_lo.append(lo)
        row_z.append(m_)
        nb += n
    if row_z and row_z[-1] - row_z[0] + 1 != len(row_z):
        raise ValueError("leaf rows of a beam are not physically adjacent (a row without beamlets in between)")
    _beam_cells.last_row_lo = row_lo                  # picked up by generate() (row_col0)
    return cell_to_bl, row_len, u0, z0


def _beam_entries(spec: PhantomSpec, theta_deg, x, y, z, target_mask, bl_base):
    """All kept (voxel, beamlet, value) entries of one beam, voxel-major with ascending beamlets."""
    th = np.deg2rad(theta_deg)
    dx, dy = np.sin(th), -np.cos(th)            # direction of travel
    ux, uy = np.cos(th), np.sin(th)             # leaf travel axis
    u = x * ux + y * uy
    ax, ay = spec.body_axes_mm
    qa = dx * dx / (ax * ax) + dy * dy / (ay * ay)
    qb = x * dx / (ax * ax) + y * dy / (ay * ay)
    qc = x * x / (ax * ax) + y * y / (ay * ay) - 1.0
    depth = (qb + np.sqrt(np.maximum(qb * qb - qa * qc, 0.0))) / qa
    cell_to_bl, row_len, u0, z0 = _beam_cells(spec, u, z, target_mask)
    ncz, ncu = cell_to_bl.shape
    bu, bz = spec.beamlet_mm
    # voxels that can see the field at all
    sel = np.nonzero((u >= u0 - WINDOW_MM) & (u <= u0 + (ncu - 1) * bu + WINDOW_MM) &
                     (z >= z0 - WINDOW_MM) & (z <= z0 + (ncz - 1) * bz + WINDOW_MM))[0]
    us, zs = u[sel].astype(np.float32), z[sel].astype(np.float32)
    att = np.exp(-MU_PER_MM * depth[sel]).astype(np.float32)
    cu = np.rint((us - u0) / bu).astype(np.int64)
    cz = np.rint((zs - z0) / bz).astype(np.int64)
    wu, wz = int(np.ceil(WINDOW_MM / bu)), int(np.ceil(WINDOW_MM / bz))
    ou = np.arange(-wu, wu + 1)
    oz = np.arange(-wz, wz + 1)
    n_sel, n_off = sel.size, ou.size * oz.size
    inv2s2 = np.float32(1.0 / (2.0 * SIGMA_MM * SIGMA_MM))
    # separable lateral Gaussian: exp(-(du^2 + dz^2)/(2 s^2)) = eu * ez
    du = (np.float32(u0) + (cu[:, None] + ou[None, :]).astype(np.float32) * np.float32(bu)) - us[:, None]
    dz = (np.float32(z0) + (cz[:, None] + oz[None, :]).astype(np.float32) * np.float32(bz)) - zs[:, None]
    eu = np.exp(-(du * du) * inv2s2)
    ez = np.exp(-(dz * dz) * inv2s2) * att[:, None]
    vals = (ez[:, :, None] * eu[:, None, :]).reshape(n_sel, n_off)        # offsets row-major (z, u)
    # beamlet id of every (voxel, offset): lookup in the cell grid padded with -1
    pu, pz = 2 * wu + 1, 2 * wz + 1
    pad = np.full((ncz + 2 * pz, ncu + 2 * pu), -1, dtype=np.int32)
    pad[pz:pz + ncz, pu:pu + ncu] = cell_to_bl
    bls = pad[(cz[:, None, None] + pz + oz[None, :, None]),
              (cu[:, None, None] + pu + ou[None, None, :])].reshape(n_sel, n_off)
    vals[bls < 0] = 0.0
    nbl = int(sum(row_len))
    # column maximum over ALL in-body voxels (those outside `sel` are far below the cut-off):
    # group voxels by base cell, one reduceat, then fold the per-(cell, offset) maxima per beamlet
    base = cz * (ncu + 2 * pu) + cu
    order = np.argsort(base, kind="stable")
    sb = base[order]
    seg = np.nonzero(np.r_[True, sb[1:] != sb[:-1]])[0]
    seg_max = np.maximum.reduceat(vals[order], seg, axis=0)                # [n_seg, n_off]
    seg_cu, seg_cz = cu[order][seg], cz[order][seg]
    seg_bl = pad[(seg_cz[:, None, None] + pz + oz[None, :, None]),
                 (seg_cu[:, None, None] + pu + ou[None, None, :])].reshape(seg.size, n_off)
    colmax = np.zeros(nbl, dtype=np.float32)
    for k in range(n_off):                       # base cells are unique within one offset
        good = seg_bl[:, k] >= 0
        b = seg_bl[good, k]
        colmax[b] = np.maximum(colmax[b], seg_max[good, k])
    thr = np.float32(REL_CUTOFF) * colmax
    keep = (bls >= 0) & (vals >= thr[np.maximum(bls, 0)])
    counts = keep.sum(axis=1).astype(np.int64)
    ent_bl = (bls[keep] + bl_base).astype(np.int32)      # row-major nonzero order = voxel-major
    ent_val = vals[keep]
    return sel, counts, ent_bl, ent_val, row_len


def generate(spec: PhantomSpec, seed: int = 0) -> Phantom:
    rng = np.random.default_rng(seed)
    lin, x, y, z = _in_body_voxels(spec)
    sid, names, tu, wu, to, wo = _assign_structures(spec, x, y, z, rng)
    tgt_ids = [i for i, st in enumerate(spec.structures) if st.is_target]
    target_mask = np.isin(sid, tgt_ids)
    if not target_mask.any():
        raise ValueError("phantom has no target voxels")
    g0 = spec.gantry_start_deg + (float(rng.uniform(0.0, 1.0)) if spec.jitter else 0.0)
    gantry = [g0 + 360.0 * b / spec.n_beams for b in range(spec.n_beams)]

    n_in = x.size
    per_beam = []
    beam_row_ptr = [0]
    row_bl_ptr = [0]
    row_col0 = []
    bl_base = 0
    total = np.zeros(n_in, dtype=np.int64)
    for th in gantry:
        sel, counts, ent_bl, ent_val, row_len = _beam_entries(spec, th, x, y, z, target_mask, bl_base)
        per_beam.append((sel, counts, ent_bl, ent_val))
        total[sel] += counts
        for n in row_len:
            row_bl_ptr.append(row_bl_ptr[-1] + n)
        lo0 = min(_beam_cells.last_row_lo)
        row_col0.extend(int(v - lo0) for v in _beam_cells.last_row_lo)
        beam_row_ptr.append(len(row_bl_ptr) - 1)
        bl_base += int(sum(row_len))
    n_bl = bl_base

    keep_vox = np.nonzero(total > 0)[0]                  # voxels with >= 1 nonzero, compact ids
    new_id = np.full(n_in, -1, dtype=np.int64)
    new_id[keep_vox] = np.arange(keep_vox.size)
    cnt = total[keep_vox]
    nnz = int(cnt.sum())
    if nnz >= 2 ** 31:
        raise ValueError("nnz >= 2^31")
    row_ptr = np.zeros(keep_vox.size + 1, dtype=np.int64)
    np.cumsum(cnt, out=row_ptr[1:])
    col_idx = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float32)
    cursor = row_ptr[:-1].copy()                         # next free slot of each voxel row
    for sel, counts, ent_bl, ent_val in per_beam:
        has = counts > 0
        rows = new_id[sel[has]]
        c = counts[has]
        start = cursor[rows]
        # position of every entry: start of its voxel's slot + rank inside the beam's run
        first = np.zeros(c.size, dtype=np.int64)
        np.cumsum(c[:-1], out=first[1:])
        pos = np.repeat(start - first, c) + np.arange(ent_bl.size, dtype=np.int64)
        col_idx[pos] = ent_bl
        val[pos] = ent_val
        cursor[rows] += c

    tgt_presc = [spec.structures[i].t_under for i in tgt_ids]
    return Phantom(
        name=spec.name, seed=seed, n_vox=int(keep_vox.size), n_bl=int(n_bl), nnz=nnz,
        row_ptr=row_ptr.astype(np.int32), col_idx=col_idx, val=val,
        n_beams=spec.n_beams, n_rows=len(row_bl_ptr) - 1,
        beam_row_ptr=np.asarray(beam_row_ptr, dtype=np.int32),
        row_bl_ptr=np.asarray(row_bl_ptr, dtype=np.int32),
        row_col0=np.asarray(row_col0, dtype=np.int32),
        n_struct=len(names), vox_struct=sid[keep_vox].astype(np.int32),
        t_under=tu, w_under=wu, t_over=to, w_over=wo, struct_names=names,
        gantry_deg=gantry, vox_grid_index=lin[keep_vox], grid=spec.grid, voxel_mm=spec.voxel_mm,
        prescription=float(max(tgt_presc)))


# --------------------------------------------------------------------------- BASELINE.json configs
def _target(name, shapes, presc):
    # targets: alpha = 10 at T^- = prescription, beta = 5 at T^+ = 1.05 * prescription (configs[0])
    return StructureSpec(name, shapes, presc, 10.0, 1.05 * presc, 5.0, is_target=True)


def _oar(name, shapes, t_over, w_over=2.0):
    return StructureSpec(name, shapes, 0.0, 0.0, t_over, w_over)


_BODY_WEAK = StructureSpec("body", [], 0.0, 0.0, 0.5, 0.5)      # reading S9: weak body penalty


def spec_tiny() -> PhantomSpec:
    """BASELINE.json configs[0]."""
    return PhantomSpec(
        name="cfg0_tiny", grid=(32, 32, 32), voxel_mm=2.5, body_axes_mm=(38.0, 38.0),
        structures=[_target("target", [Shape("ellipsoid", (0, 0, 0), (12, 12, 12))], 1.0),
                    _oar("oar", [Shape("ellipsoid", (0, 18, 0), (8, 8, 8))], 0.3)],
        body=None, n_beams=1, beamlet_mm=(5.0, 5.0), field="fixed", fixed_grid=(10, 10),
        gantry_start_deg=0.0, jitter=False)


def spec_prostate(ptv_scale: float = 2.0, n_beams: int = 9, voxel_mm: float = 2.5,
                  grid=(200, 200, 120), beamlet_mm=(5.0, 5.0), name: Optional[str] = None) -> PhantomSpec:
    """BASELINE.json configs[1] (9 fields, 2.5 mm) and configs[4] (7 fields, 2.0 mm, 2.5x5 beamlets).

    ptv_scale multiplies the PTV semi-axes (30, 25, 30) mm; the literal geometry (scale 1) gives
    about 3x fewer beamlets / non-zeros than BASELINE.json's own "about 30x24 per beam, 30-60M
    nnz"; scale 2 lands inside that band.  OARs move with the PTV surface."""
    s = ptv_scale
    px, py, pz = 30.0 * s, 25.0 * s, 30.0 * s
    return PhantomSpec(
        name=name or f"prostate_{n_beams}f_x{ptv_scale:g}", grid=grid, voxel_mm=voxel_mm,
        body_axes_mm=(180.0, 110.0),
        structures=[
            _target("ptv", [Shape("ellipsoid", (0, 0, 0), (px, py, pz))], 1.0),
            _oar("rectum", [Shape("zcyl", (0, -(py + 10.0), 0), (10.0, 0, pz))], 0.5),
            _oar("bladder", [Shape("ellipsoid", (0, py + 12.0, pz * 0.5 + 15.0), (30, 30, 30))], 0.5),
            _oar("femur_l", [Shape("ellipsoid", (-90 - 10 * (s - 1), 0, 0), (22, 22, 22))], 0.3),
            _oar("femur_r", [Shape("ellipsoid", (90 + 10 * (s - 1), 0, 0), (22, 22, 22))], 0.3),
        ],
        body=_BODY_WEAK, n_beams=n_beams, beamlet_mm=beamlet_mm, field="ptv")


def spec_headneck(scale: float = 1.0, name: Optional[str] = None) -> PhantomSpec:
    """BASELINE.json configs[2]: 5 fields, union-of-3-ellipsoids PTV1 (1.0), spherical PTV2 (0.85)."""
    s = scale
    return PhantomSpec(
        name=name or f"headneck_5f_x{scale:g}", grid=(256, 256, 160), voxel_mm=2.5,
        body_axes_mm=(90.0, 110.0),
        structures=[
            _target("ptv1", [Shape("ellipsoid", (-20 * s, 10, 10 * s), (45 * s, 35, 50 * s)),
                             Shape("ellipsoid", (25 * s, 20, -15 * s), (40 * s, 30, 45 * s)),
                             Shape("ellipsoid", (0, -5, 40 * s), (35 * s, 30, 35 * s))], 1.0),
            _target("ptv2", [Shape("ellipsoid", (35 * s, -20, -55 * s), (25, 25, 25))], 0.85),
            _oar("cord", [Shape("zcyl", (0, -60, 0), (6.0, 0, 150.0))], 0.45),
            _oar("parotid_l", [Shape("ellipsoid", (-68, 5, 20), (12, 18, 22))], 0.3),
            _oar("parotid_r", [Shape("ellipsoid", (68, 5, 20), (12, 18, 22))], 0.3),
            _oar("brainstem", [Shape("ellipsoid", (0, -35, 95), (14, 14, 18))], 0.5),
        ],
        body=_BODY_WEAK, n_beams=5, beamlet_mm=(5.0, 5.0), field="ptv")


def spec_stress(ptv_scale: float = 2.2) -> PhantomSpec:
    """BASELINE.json configs[4]: 7-field prostate shape, 2.0 mm voxels, 2.5 x 5 mm beamlets."""
    return spec_prostate(ptv_scale=ptv_scale, n_beams=7, voxel_mm=2.0, grid=(250, 250, 150),
                         beamlet_mm=(2.5, 5.0), name=f"stress_7f_x{ptv_scale:g}")


def spec_mini(n_beams: int = 3, ptv_scale: float = 0.8) -> PhantomSpec:
    """A small multi-beam prostate-shaped case for parity tests (seconds in the oracle)."""
    sp = spec_prostate(ptv_scale=ptv_scale, n_beams=n_beams, voxel_mm=5.0, grid=(80, 52, 24),
                       name=f"mini_{n_beams}f")
    return sp


CONFIGS = {
    "cfg0": spec_tiny,
    "cfg1": lambda: spec_prostate(2.0),
    "cfg1_literal": lambda: spec_prostate(1.0),
    "cfg2": lambda: spec_headneck(1.8),          # fields of about 40x30 beamlets, as configs[2] states
    "cfg2_literal": lambda: spec_headneck(1.0),
    "cfg4": lambda: spec_stress(2.2),
    "cfg4_literal": lambda: spec_stress(1.0),
    "mini": spec_mini,
    # the paper's own problem size (Table 1: case P1 has 7,196 beamlets, 45,912 voxels, 2.76M
    # non-zeros; unspecified tissue at coarse resolution): 9 fields, 6.5 mm voxels -> 7,337 beamlets, 42,898 voxels, 4.5M
    "paper_p1": lambda: spec_prostate(2.7, n_beams=9, voxel_mm=6.5, grid=(70, 44, 32), name="paper_p1"),
    # BASELINE.json configs[3] (kernel sweep): pencil-beam matrices from ~1M to ~200M non-zeros
    "sweep_1m": lambda: spec_prostate(1.0, n_beams=5, voxel_mm=4.0, grid=(126, 126, 76), name="sweep_1m"),
    "sweep_3m": lambda: spec_prostate(1.0, n_beams=9, voxel_mm=4.0, grid=(126, 126, 76), name="sweep_3m"),
    "sweep_100m": lambda: spec_stress(1.7),
    "sweep_200m": lambda: spec_stress(2.4),
}


def make(config: str, seed: int = 0) -> Phantom:
    """``config`` is a key of CONFIGS, optionally followed by ``_reopt`` (re-optimisation mode)."""
    if config.endswith("_reopt"):
        return reoptimisation(generate(CONFIGS[config[:-6]](), seed), seed)
    return generate(CONFIGS[config](), seed)


# --------------------------------------------------------------------------- re-optimisation inputs
def reoptimisation(ph: Phantom, seed: int = 0, falloff_mm: float = 25.0, shift_mm: float = 4.0,
                   ripple: float = 0.03) -> Phantom:
    """The same geometry posed as the paper's re-optimisation problem: alpha_j =
    beta_j = 1, T_j = "the dose distribution from the original plan, deformed to the daily image".

    The clinical reference doses are not available, so T_j is a smooth synthetic stand-in with the
    shape of a delivered plan: the prescription inside a target-sized ball around the (shifted)
    target centroid, an exponential fall-off with distance outside it, and a seeded low-frequency
    ripple (the "deformation").  Structures become 0 = target voxels (under- and over-dose
    penalised, eq. 3-4) and 1 = all other voxels (over-dose only).  No method arithmetic here."""
    rng = np.random.default_rng(seed + 7919)
    nx, ny, nz = ph.grid
    lin = ph.vox_grid_index
    ix, iy, iz = lin % nx, (lin // nx) % ny, lin // (nx * ny)
    h = ph.voxel_mm
    x = (ix - (nx - 1) / 2.0) * h
    y = (iy - (ny - 1) / 2.0) * h
    z = (iz - (nz - 1) / 2.0) * h
    is_target = np.zeros(ph.n_vox, dtype=bool)
    for s in range(ph.n_struct):
        if ph.w_under[s] > 0:
            is_target |= ph.vox_struct == s
    c = np.array([x[is_target].mean(), y[is_target].mean(), z[is_target].mean()])
    c = c + rng.uniform(-shift_mm, shift_mm, size=3)
    radius = (3.0 * is_target.sum() * h ** 3 / (4.0 * np.pi)) ** (1.0 / 3.0)
    d = np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)
    t = ph.prescription * np.exp(-np.maximum(d - radius, 0.0) / falloff_mm)
    ph_x, ph_y, ph_z = rng.uniform(0.0, 2.0 * np.pi, size=3)
    t = t * (1.0 + ripple * np.sin(x / 37.0 + ph_x) * np.sin(y / 41.0 + ph_y) * np.sin(z / 29.0 + ph_z))
    import copy
    q = copy.copy(ph)
    q.name = ph.name + "_reopt"
    q.n_struct = 2
    q.vox_struct = np.where(is_target, 0, 1).astype(np.int32)
    q.t_under = np.zeros(2, dtype=np.float32)
    q.t_over = np.zeros(2, dtype=np.float32)
    q.w_under = np.array([1.0, 0.0], dtype=np.float32)
    q.w_over = np.array([1.0, 1.0], dtype=np.float32)
    q.struct_names = ["target", "other"]
    q.vox_threshold = t.astype(np.float32)
    q.per_voxel_weights = True
    return q


# --------------------------------------------------------------------------- kernel-sweep inputs
def pricing_rows(n_rows: int, row_len: int, rows_per_beam: int, seed: int = 0):
    """configs[3] pricing sweep: i.i.d. N(0,1) beamlet gradients plus a smooth negative bump per
    beam; returns (w float32 [n_rows*row_len], beam_row_ptr, row_bl_ptr)."""
    rng = np.random.default_rng(seed)
    n_beams = (n_rows + rows_per_beam - 1) // rows_per_beam
    w = rng.standard_normal((n_rows, row_len))
    m = np.arange(n_rows) % rows_per_beam
    b = np.arange(n_rows) // rows_per_beam
    c0 = rng.uniform(0, row_len, size=n_beams)[b]
    m0 = rng.uniform(0, rows_per_beam, size=n_beams)[b]
    s = row_len / 4.0
    c = np.arange(row_len)[None, :]
    w -= 2.0 * np.exp(-((c - c0[:, None]) ** 2 + (m[:, None] - m0[:, None]) ** 2) / (2 * s * s))
    beam_row_ptr = np.minimum(np.arange(n_beams + 1) * rows_per_beam, n_rows).astype(np.int32)
    row_bl_ptr = (np.arange(n_rows + 1) * row_len).astype(np.int32)
    return w.astype(np.float32).ravel(), beam_row_ptr, row_bl_ptr


def random_csr(n_rows: int, n_cols: int, density: float, seed: int = 0, empty_rows: bool = True):
    """Small random CSR (fp32/int32, ascending columns) for unit tests, incl. empty rows/columns."""
    rng = np.random.default_rng(seed)
    mask = rng.random((n_rows, n_cols)) < density
    if empty_rows and n_rows > 2:
        mask[rng.integers(0, n_rows)] = False
    if empty_rows and n_cols > 2:
        mask[:, rng.integers(0, n_cols)] = False
    dense = np.where(mask, rng.random((n_rows, n_cols)).astype(np.float32), np.float32(0))
    row_ptr = np.zeros(n_rows + 1, dtype=np.int32)
    row_ptr[1:] = np.cumsum(mask.sum(axis=1))
    r, c = np.nonzero(mask)
    return row_ptr, c.astype(np.int32), dense[r, c].astype(np.float32), dense
