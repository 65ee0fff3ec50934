"""Host logic of the voxel-row sharding slice (paper_1003_5402_b200/sharded.py) on CPU: the partition,
the slab view of a problem, the rank-ordered reduction -- alone and across two processes over gloo (127.0.0.1).
The arithmetic used to check it is test-local numpy (dense products on the tiny instance)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1003_5402_b200 import sharded

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _dense(ph):
    A = np.zeros((ph.n_vox, ph.n_bl))
    for v in range(ph.n_vox):
        s, e = ph.row_ptr[v], ph.row_ptr[v + 1]
        A[v, ph.col_idx[s:e]] = ph.val[s:e]
    return A


@pytest.mark.parametrize("world", [1, 2, 3, 7])
@pytest.mark.parametrize("balance", [False, True])
def test_slab_bounds_tile_the_voxels(tiny, world, balance):
    b = sharded.slab_bounds(tiny.n_vox, world, tiny.row_ptr if balance else None)
    assert len(b) == world and b[0][0] == 0 and b[-1][1] == tiny.n_vox
    assert all(b[i][1] == b[i + 1][0] for i in range(world - 1)) and all(v0 <= v1 for v0, v1 in b)
    if balance and world > 1:
        nnz = [int(tiny.row_ptr[v1] - tiny.row_ptr[v0]) for v0, v1 in b]
        longest = int(np.diff(tiny.row_ptr).max())
        assert max(nnz) - min(nnz) <= 2 * longest + 1          # cut points land on row boundaries


def test_more_ranks_than_voxels_gives_empty_slabs():
    b = sharded.slab_bounds(3, 5)
    assert sum(v1 - v0 for v0, v1 in b) == 3 and len(b) == 5


def test_slabs_reassemble_the_problem(tiny):
    A = _dense(tiny)
    rng = np.random.default_rng(3)
    x, g = rng.random(tiny.n_bl), rng.standard_normal(tiny.n_vox)
    z_parts, w_parts = [], []
    count = np.bincount(tiny.vox_struct[tiny.vox_struct >= 0], minlength=len(tiny.t_under))
    for v0, v1 in sharded.slab_bounds(tiny.n_vox, 3, tiny.row_ptr):
        s = sharded.make_slab(tiny, v0, v1)
        assert s.n_vox == v1 - v0 and s.row_ptr[0] == 0 and s.row_ptr[-1] == s.nnz == s.col_idx.size == s.val.size
        assert np.array_equal(s.struct_count, count)                 # |v_s| of the WHOLE problem on every slab
        As = _dense(s)
        assert np.array_equal(As, A[v0:v1])
        z_parts.append(As @ x)
        w_parts.append(As.T @ g[v0:v1])
    assert np.allclose(np.concatenate(z_parts), A @ x, rtol=0, atol=1e-14)
    assert np.allclose(sharded.sum_in_rank_order(w_parts), A.T @ g, rtol=1e-13, atol=1e-13)


def test_sum_in_rank_order_is_the_left_to_right_sum():
    parts = [np.array([1e16, 1.0]), np.array([-1e16, 1.0]), np.array([1.0, 1e-20])]
    assert np.array_equal(sharded.sum_in_rank_order(parts), (parts[0] + parts[1]) + parts[2])


def test_all_reduce_without_process_group_is_identity():
    v = np.arange(5, dtype=np.float32)
    out = sharded.all_reduce_in_rank_order(v)
    assert out.dtype == np.float64 and np.array_equal(out, v)


WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np
import torch.distributed as dist
from paper_1003_5402_b200 import sharded
from conftest import TinyCase
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ph = TinyCase(seed=1)
v0, v1 = sharded.slab_bounds(ph.n_vox, world, ph.row_ptr)[rank]
s = sharded.make_slab(ph, v0, v1)
g = np.random.default_rng(5).standard_normal(ph.n_vox)      # the same vector on every rank
w_r = np.zeros(ph.n_bl)
for v in range(s.n_vox):                                      # this rank's partial sum of D^T g (eq. 8)
    a, b = s.row_ptr[v], s.row_ptr[v + 1]
    np.add.at(w_r, s.col_idx[a:b], s.val[a:b].astype(np.float64) * g[v0 + v])
w = sharded.all_reduce_in_rank_order(w_r)
json.dump({{"rank": rank, "v0": v0, "v1": v1, "w": w.tolist()}}, open(os.path.join({out!r}, f"r{{rank}}.json"), "w"))
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_over_gloo_hold_the_same_gradient(tiny, tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.load(open(tmp_path / f"r{i}.json")) for i in range(2)]
    assert res[0]["v0"] == 0 and res[0]["v1"] == res[1]["v0"] and res[1]["v1"] == tiny.n_vox
    assert res[0]["w"] == res[1]["w"]                                  # bit-identical on both ranks
    g = np.random.default_rng(5).standard_normal(tiny.n_vox)
    assert np.allclose(res[0]["w"], _dense(tiny).T @ g, rtol=1e-12, atol=1e-12)
