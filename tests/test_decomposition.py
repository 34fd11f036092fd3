"""Host logic of the brick decomposition: the arithmetic of
`BrickDecomposition` and the halo exchange `exchange_layers` over two gloo ranks on the CPU.  (The packing of a layer and the
sweeps that read it are CUDA: tests/test_gpu_parity.py::test_brick_decomposition_* checks decomposed == undivided, bit for
bit, on a B200.)"""
import itertools
import json
import os
import socket
import subprocess
import sys

import pytest

from paper_1810_13416_b200.decomposition import BC_HALO, BC_PERIODIC, BC_REFLECT, BrickDecomposition

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
P, R, H = BC_PERIODIC, BC_REFLECT, BC_HALO


def test_subdomains_tile_the_grid_and_ranks_round_trip():
    d = BrickDecomposition((64, 32, 48), (2, 1, 3), (R,) * 6)
    assert d.size == 6 and d.local_n() == (32, 32, 16)
    seen = set()
    for r in range(d.size):
        assert d.rank_of(d.coords(r)) == r
        org = d.origin(r)
        for c in itertools.product(*[range(org[k], org[k] + d.local_n()[k], 8) for k in range(3)]):
            assert c not in seen
            seen.add(c)
    assert len(seen) == (64 // 8) * (32 // 8) * (48 // 8)


def test_neighbours_are_mutual_and_walls_have_none():
    d = BrickDecomposition((64, 64, 64), (2, 2, 2), (R, R, P, P, R, R))
    for r in range(8):
        for axis in range(3):
            for side in (0, 1):
                q = d.neighbour(r, axis, side)
                if q is not None:
                    assert d.neighbour(q, axis, 1 - side) == r
        c = d.coords(r)
        # x, z: walls of the global grid stay walls; y: periodic, every sub-domain has both neighbours (the same rank twice)
        assert d.local_bc(r) == (R if c[0] == 0 else H, R if c[0] == 1 else H, H, H, R if c[2] == 0 else H, R if c[2] == 1 else H)
        assert d.neighbour(r, 1, 0) == d.neighbour(r, 1, 1) != r
    # an axis that is not cut keeps its boundary types (a periodic one wraps inside the library)
    d1 = BrickDecomposition((32, 32, 64), (1, 1, 2), (P, P, R, R, P, P))
    assert d1.local_bc(0) == (P, P, R, R, H, H) and d1.neighbour(0, 0, 0) is None


def test_bad_splits_are_refused():
    with pytest.raises(ValueError):
        BrickDecomposition((60, 64, 64), (2, 1, 1), (R,) * 6)        # 30 cells per sub-domain: not whole bricks
    with pytest.raises(ValueError):
        BrickDecomposition((8, 64, 64), (2, 1, 1), (R,) * 6)         # one brick per sub-domain: the two halos would overlap
    with pytest.raises(ValueError):
        BrickDecomposition((64, 64, 64), (2, 1, 1), (P, R, R, R, R, R))
    assert BrickDecomposition((64, 64, 64), (1, 1, 1), (R,) * 6).local_bc(0) == (R,) * 6


def test_exchange_plans_match_pairwise_in_posting_order():
    """every send has its receive, and between any two ranks the k-th message sent is the k-th received with the side swapped
    (NCCL matches in posting order) — also when both neighbours are the same rank"""
    for procs, bc in (((2, 2, 2), (R,) * 6), ((2, 1, 1), (P, P, R, R, R, R)), ((4, 1, 2), (P, P, R, R, P, P)), ((3, 1, 1), (P, P, R, R, R, R))):
        d = BrickDecomposition((96, 32, 32), procs, bc)
        for axis in range(3):
            plans = {r: d.exchange_plan(r, axis) for r in range(d.size)}
            for r in range(d.size):
                for q in range(d.size):
                    sends = [side for kind, peer, side in plans[r] if kind == "send" and peer == q]
                    recvs = [side for kind, peer, side in plans[q] if kind == "recv" and peer == r]
                    assert [1 - s for s in sends] == recvs, (procs, axis, r, q, sends, recvs)
            n_faces = sum(1 for r in range(d.size) for s in (0, 1) if d.neighbour(r, axis, s) is not None)
            assert sum(len(p) for p in plans.values()) == 2 * n_faces
        assert d.halo_cells(0) == 4 * d.local_n()[1] * d.local_n()[2]


WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch
import torch.distributed as dist
from paper_1810_13416_b200.decomposition import BrickDecomposition, exchange_layers
rank, ws = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=ws)
ok = {}
for name, n, procs, bc, axis in (("walls", (16, 8, 8), (2, 1, 1), (1,) * 6, 0), ("periodic", (8, 8, 32), (1, 1, 2), (1, 1, 1, 1, 0, 0), 2)):
    d = BrickDecomposition(n, procs, bc)
    # a global array every rank can rebuild: value = global cell index; layers packed by slicing (the CPU stand-in for
    # ppm_pack_halo: 4 cells deep, all cells of the two other axes)
    g = np.arange(n[0] * n[1] * n[2], dtype=np.float32).reshape(n[2], n[1], n[0])
    def box(r):
        o, ln = d.origin(r), d.local_n()
        return g[o[2]:o[2] + ln[2], o[1]:o[1] + ln[1], o[0]:o[0] + ln[0]]
    def layer(r, side):
        b = np.moveaxis(box(r), 2 - axis, 0)          # the sweep axis first
        return np.ascontiguousarray(b[-4:] if side else b[:4])
    send = {s: torch.from_numpy(layer(rank, s).copy()) for s in (0, 1)}
    recv = {s: torch.full_like(send[s], -1.0) for s in (0, 1)}
    exchange_layers(d, rank, axis, send, recv)
    good = True
    for s in (0, 1):
        q = d.neighbour(rank, axis, s)
        if q is None:
            good &= bool((recv[s] == -1.0).all())                          # a wall: nothing arrives
        else:
            good &= bool(np.array_equal(recv[s].numpy(), layer(q, 1 - s)))    # the neighbour's layer that touches this face
    ok[name] = good
# the two scalar reductions of a decomposed step
t = torch.tensor([0.5 + rank], dtype=torch.float64); dist.all_reduce(t, op=dist.ReduceOp.MIN); ok["dt"] = float(t) == 0.5
t = torch.tensor([1.0 + rank] * 6, dtype=torch.float64); dist.all_reduce(t, op=dist.ReduceOp.SUM); ok["sum"] = t.tolist() == [3.0] * 6
print(json.dumps(ok))
dist.barrier()
dist.destroy_process_group()
"""


def test_halo_exchange_two_gloo_ranks_walls_and_periodic_wrap():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for o in outs:
        res = json.loads(o[0].strip().splitlines()[-1])
        assert res == {"walls": True, "periodic": True, "dt": True, "sum": True}, res
