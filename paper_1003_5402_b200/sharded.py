"""Voxel-row sharding of the column-generation iteration, first slice (the paper itself runs on one
GPU).

Rank r of R owns a contiguous slab of the voxel rows of D, with it the slab's part of z, pi and of every
aperture-dose column.  Steps 2 and 3 (dose, objective, voxel gradient) are local; step 4
(eq. 8) becomes the slab's partial sum ``w_r = D_r^T pi_r`` followed by ONE all-reduce of
N values per column-generation iteration; steps 5 and 6 (pricing) run replicated on the summed
``w``; step 7 (eq. 2) is local again.  The only thing a slab context must be told is |v_s| of the WHOLE problem
(eq. 9-10 normalise by it): ``dao_structs.struct_count``.

This module holds the host logic only -- the partition, the slab view of a problem, the fixed-order reduction --
and marshals; every product runs in the kernels of libdao.so through :class:`paper_1003_5402_b200.dao.Dao`.  The
restricted master (step 8) is not sharded here: it needs the (H, gradient, F) block summed over the ranks once
per pass INSIDE the persistent kernel.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np


def slab_bounds(n_vox: int, world_size: int, row_ptr: Optional[np.ndarray] = None) -> List[Tuple[int, int]]:
    """Contiguous voxel ranges, one per rank.  With ``row_ptr`` the cut points balance the NON-ZEROS (what the
    SpMVs stream), otherwise the voxels; every rank gets a (possibly empty) range, the ranges tile [0, n_vox)."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    if row_ptr is None:
        cuts = [(n_vox * r) // world_size for r in range(world_size + 1)]
    else:
        rp = np.asarray(row_ptr, dtype=np.int64)
        nnz = int(rp[-1])
        cuts = [0]
        for r in range(1, world_size):
            cuts.append(int(np.searchsorted(rp, (nnz * r) // world_size, side="left")))
        cuts.append(n_vox)
        cuts = [min(max(c, 0), n_vox) for c in cuts]
        for i in range(1, len(cuts)):
            cuts[i] = max(cuts[i], cuts[i - 1])
    return [(cuts[r], cuts[r + 1]) for r in range(world_size)]


@dataclass
class Slab:
    """The fields :class:`paper_1003_5402_b200.dao.Dao` reads, restricted to the voxel rows [v0, v1)."""
    name: str
    v0: int
    v1: int
    n_vox: int
    n_bl: int
    nnz: int
    row_ptr: np.ndarray
    col_idx: np.ndarray
    val: np.ndarray
    n_beams: int
    n_rows: int
    beam_row_ptr: np.ndarray
    row_bl_ptr: np.ndarray
    n_struct: int
    vox_struct: np.ndarray
    t_under: np.ndarray
    w_under: np.ndarray
    t_over: np.ndarray
    w_over: np.ndarray
    struct_count: np.ndarray                 # int64 [n_struct]: |v_s| of the WHOLE problem
    prescription: float = 1.0
    vox_threshold: Optional[np.ndarray] = None
    per_voxel_weights: bool = False
    row_col0: Optional[np.ndarray] = None


def make_slab(ph, v0: int, v1: int) -> Slab:
    """Rows [v0, v1) of the problem ``ph`` (views, no copies of the matrix)."""
    if not (0 <= v0 <= v1 <= ph.n_vox):
        raise ValueError("bad slab range")
    rp = np.asarray(ph.row_ptr)
    e0, e1 = int(rp[v0]), int(rp[v1])
    vs = np.asarray(ph.vox_struct)
    count = np.bincount(vs[vs >= 0], minlength=int(ph.n_struct)).astype(np.int64)
    vt = getattr(ph, "vox_threshold", None)
    return Slab(name=f"{ph.name}[{v0}:{v1}]", v0=v0, v1=v1, n_vox=v1 - v0, n_bl=int(ph.n_bl), nnz=e1 - e0,
                row_ptr=(rp[v0:v1 + 1] - rp[v0]).astype(np.int32), col_idx=ph.col_idx[e0:e1], val=ph.val[e0:e1],
                n_beams=int(ph.n_beams), n_rows=int(ph.n_rows), beam_row_ptr=ph.beam_row_ptr, row_bl_ptr=ph.row_bl_ptr,
                n_struct=int(ph.n_struct), vox_struct=vs[v0:v1], t_under=ph.t_under, w_under=ph.w_under,
                t_over=ph.t_over, w_over=ph.w_over, struct_count=count, prescription=float(getattr(ph, "prescription", 1.0)),
                vox_threshold=None if vt is None else np.asarray(vt)[v0:v1],
                per_voxel_weights=bool(getattr(ph, "per_voxel_weights", False)), row_col0=getattr(ph, "row_col0", None))


def sum_in_rank_order(parts: Sequence[np.ndarray]) -> np.ndarray:
    """fp64 sum of the ranks' shares in rank order: the same bits whatever the arrival order."""
    acc = np.zeros_like(np.asarray(parts[0], dtype=np.float64))
    for p in parts:
        acc = acc + np.asarray(p, dtype=np.float64)
    return acc


def all_reduce_in_rank_order(local: np.ndarray, group=None) -> np.ndarray:
    """The all-reduce of step 4 over ``torch.distributed`` (NCCL between GPUs, gloo on CPU): every rank gathers
    every share and adds them in rank order, so that all ranks hold bit-identical ``w`` (pricing is replicated and
    must take the same decision everywhere).  N values per column-generation iteration: latency, not bandwidth."""
    import torch
    import torch.distributed as dist

    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return np.asarray(local, dtype=np.float64).copy()
    backend = dist.get_backend(group)
    dev = "cuda" if backend == "nccl" else "cpu"
    mine = torch.from_numpy(np.ascontiguousarray(local, dtype=np.float64)).to(dev)
    parts = [torch.empty_like(mine) for _ in range(dist.get_world_size(group))]
    dist.all_gather(parts, mine, group=group)
    return sum_in_rank_order([p.cpu().numpy() for p in parts])


class ShardedIteration:
    """Steps 2-6 of one column-generation iteration on this rank's slab.  ``dao`` is the module
    :mod:`paper_1003_5402_b200.dao`; one context per rank, created on the slab with the global |v_s|."""

    def __init__(self, dao, ph, rank: int, world_size: int, balance_nnz: bool = True, **options):
        self.rank, self.world_size = rank, world_size
        self.bounds = slab_bounds(int(ph.n_vox), world_size, ph.row_ptr if balance_nnz else None)
        v0, v1 = self.bounds[rank]
        self.slab = make_slab(ph, v0, v1)
        self._dao = dao
        self.ctx = dao.Dao(self.slab, **options)

    def close(self):
        self.ctx.close()

    def local_shares(self, x_dev):
        """(F_r, w_r): this slab's share of the objective and of w = D^T pi at the beamlet intensities x
        (a CUDA float32 tensor of n_bl values, the same on every rank)."""
        f_r = self.ctx.eval_x(x_dev)                       # dose, objective share, pi of the slab
        import torch
        g = torch.from_numpy(self.ctx.get_vector(self._dao.VEC_G)).cuda()
        w_r = self.ctx.spmv_t(g).cpu().numpy().astype(np.float64)
        return float(f_r), w_r

    def gradient(self, x_dev, group=None):
        """(F, w) of the whole problem: local shares, then the rank-ordered all-reduce (N + 1 values)."""
        f_r, w_r = self.local_shares(x_dev)
        tot = all_reduce_in_rank_order(np.r_[w_r, f_r], group)
        return float(tot[-1]), tot[:-1]

    def price(self, w: np.ndarray):
        """Steps 5-6 replicated on the summed gradient (fp32, as the unsharded path stores it)."""
        import torch
        return self.ctx.price_from_w(torch.from_numpy(np.asarray(w, dtype=np.float32)).cuda())
