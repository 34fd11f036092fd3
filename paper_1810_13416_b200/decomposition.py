"""Brick decomposition of one grid over several GPUs (MPI bricks with a halo
one briquette = 4 cells thick).  One process per GPU, `torch.distributed` (NCCL over NVLink) for the plumbing.

Design (B200-first, not the paper's): a 1-D sweep along an axis only ever needs ghost cells ALONG that axis, 4 deep = one
brick layer of whole brick records.  So instead of one (M+2)^3 - M^3 halo exchange per step paid for by redundantly updating
ghost briquettes in the earlier passes, a sub-domain exchanges, before each of the three sweeps of a step, only
its first and last brick layer along THAT sweep's axis with its two face neighbours: no edge or corner data, no redundant
ghost update, three small messages per step instead of one large one (NVLink latency is microseconds; a 512^3 sub-domain
sends 2 x 63 MB per sweep = 0.15 ms at 900 GB/s against 4.5 ms of sweep).  The library packs a layer (ppm_pack_halo), the
layer travels (here), the neighbour's sweep reads it as its ghost brick (ppm_set_halo, boundary type PPM_BC_HALO).  The
decomposed run is bit for bit the undivided one (tests/test_gpu_parity.py::test_brick_decomposition_*).

This module is argument marshalling and message plumbing only: `BrickDecomposition` is pure host arithmetic (tested on CPU),
`exchange_layers` moves tensors between ranks (tested with gloo, world size 2), `DecomposedPPM` wires both to a `PPM`
context.  `LocalCluster` runs all sub-domains of a decomposition in ONE process on one GPU (device copies instead of
messages; the kernels of different sub-domains never wait on one another) — the way the path is tested where only one GPU
is to be had.
"""
from __future__ import annotations

import numpy as np
import torch

BC_PERIODIC, BC_REFLECT, BC_HALO = 0, 1, 2
ORDERS = ((0, 1, 2), (0, 2, 1), (1, 0, 2), (1, 2, 0), (2, 0, 1), (2, 1, 0))      # ppm_step's sweep orders


class BrickDecomposition:
    """n = global cells (nx, ny, nz), procs = sub-domains per axis (px, py, pz), bc = the six global boundary types.
    Sub-domains are equal boxes; rank = (cz * py + cy) * px + cx."""

    def __init__(self, n, procs, bc):
        self.n = tuple(int(v) for v in n)
        self.procs = tuple(int(v) for v in procs)
        self.bc = tuple(int(v) for v in bc)
        if len(self.n) != 3 or len(self.procs) != 3 or len(self.bc) != 6:
            raise ValueError("need n[3], procs[3], bc[6]")
        for d in range(3):
            if self.procs[d] < 1:
                raise ValueError("procs must be >= 1")
            if self.procs[d] > 1:
                if self.n[d] % (4 * self.procs[d]) != 0 or self.n[d] // self.procs[d] < 8:
                    raise ValueError("axis %d: %d cells do not split into %d sub-domains of whole bricks (>= 2 bricks each)"
                                     % (d, self.n[d], self.procs[d]))
            if (self.bc[2 * d] == BC_PERIODIC) != (self.bc[2 * d + 1] == BC_PERIODIC):
                raise ValueError("periodic faces must pair up")
        self.size = self.procs[0] * self.procs[1] * self.procs[2]

    def coords(self, rank):
        px, py, _ = self.procs
        return (rank % px, (rank // px) % py, rank // (px * py))

    def rank_of(self, c):
        px, py, _ = self.procs
        return (c[2] * py + c[1]) * px + c[0]

    def local_n(self, rank=0):
        return tuple(self.n[d] // self.procs[d] for d in range(3))

    def origin(self, rank):
        c, ln = self.coords(rank), self.local_n()
        return tuple(c[d] * ln[d] for d in range(3))

    def neighbour(self, rank, axis, side):
        """rank beyond the low (side 0) / high (side 1) face along axis; None at a wall of the global grid or when the
        axis is not cut (a periodic axis with one sub-domain wraps onto itself inside the library)"""
        if self.procs[axis] == 1:
            return None
        c = list(self.coords(rank))
        c[axis] += 1 if side else -1
        if c[axis] < 0 or c[axis] >= self.procs[axis]:
            if self.bc[2 * axis] != BC_PERIODIC:
                return None
            c[axis] %= self.procs[axis]
        return self.rank_of(c)

    def local_bc(self, rank):
        """the six boundary types of the sub-domain: PPM_BC_HALO wherever a neighbour exists"""
        return tuple(BC_HALO if self.neighbour(rank, k // 2, k % 2) is not None else self.bc[k] for k in range(6))

    def halo_cells(self, axis):
        """cells in one exchanged layer (4 deep) of a sub-domain"""
        ln = self.local_n()
        return 4 * ln[(axis + 1) % 3] * ln[(axis + 2) % 3]

    def exchange_plan(self, rank, axis):
        """[(kind, peer, my_side)]: what this rank posts before a sweep along axis, in the order every rank uses —
        sends first (low layer, then high layer), then the receives in the order the peers' sends arrive when both
        neighbours are the same rank (two sub-domains on a periodic axis): the peer's LOW layer is my HIGH halo."""
        plan = []
        for side in (0, 1):
            p = self.neighbour(rank, axis, side)
            if p is not None:
                plan.append(("send", p, side))
        for side in (1, 0):
            p = self.neighbour(rank, axis, side)
            if p is not None:
                plan.append(("recv", p, side))
        return plan


def exchange_layers(decomp, rank, axis, send, recv, group=None):
    """One halo exchange along `axis` over torch.distributed.  send[side] = this rank's packed low / high layer, recv[side] =
    the buffer its sweeps read as the ghost brick beyond that face (tensors on the backend's device: CUDA for NCCL, CPU for
    gloo; entries for faces without a neighbour are ignored).  A layer sent from my side s arrives in the peer's halo of side
    1 - s; tags say which (NCCL ignores them and matches in posting order, which `exchange_plan` keeps consistent)."""
    import torch.distributed as dist
    ops = []
    for kind, peer, side in decomp.exchange_plan(rank, axis):
        if kind == "send":
            ops.append(dist.P2POp(dist.isend, send[side], peer, group=group, tag=2 * axis + side))
        else:
            ops.append(dist.P2POp(dist.irecv, recv[side], peer, group=group, tag=2 * axis + (1 - side)))
    if ops:
        for r in dist.batch_isend_irecv(ops):
            r.wait()


class DecomposedPPM:
    """The sub-domain of one rank: a PPM context with PPM_BC_HALO faces, its send / receive layers, and the step driven sweep
    by sweep with an exchange before each.  `exchange(axis, send, recv)` moves the layers: exchange_layers over
    torch.distributed by default, device copies inside a LocalCluster."""

    def __init__(self, decomp, rank, dx, gamma, grav=None, rho_floor=1e-10, p_floor=1e-10, device="cuda:0", exchange=None,
                 group=None):
        from .binding import PPM
        self.decomp, self.rank, self.group = decomp, rank, group
        ln, self.org = decomp.local_n(), decomp.origin(rank)
        self.ppm = PPM(ln[0], ln[1], ln[2], dx, gamma, decomp.local_bc(rank), grav, rho_floor, p_floor, device)
        self.ppm.set_origin(self.org)
        self.send, self.recv = {}, {}
        for axis in range(3):
            for side in (0, 1):
                if decomp.neighbour(rank, axis, side) is not None:
                    nfl = self.ppm.halo_floats(axis)
                    self.send[(axis, side)] = torch.empty(nfl, dtype=torch.float32, device=self.ppm.device)
                    self.recv[(axis, side)] = torch.empty(nfl, dtype=torch.float32, device=self.ppm.device)
                    self.ppm.set_halo(axis, side, self.recv[(axis, side)])
        self._exchange = exchange if exchange is not None else self._dist_exchange
        self.halo_bytes = 0          # bytes this rank has sent so far

    # ---- state in / out: the sub-domain's own box of the global arrays ----
    def box(self):
        ln = self.decomp.local_n()
        return tuple(slice(self.org[d], self.org[d] + ln[d]) for d in range(3))

    def set_state_from_global(self, fields):
        """fields: the GLOBAL [15, nz, ny, nx] array (torch or numpy); this rank loads its own box"""
        bx, by, bz = self.box()
        f = fields[:, bz, by, bx]
        f = torch.as_tensor(np.ascontiguousarray(f) if isinstance(f, np.ndarray) else f.contiguous())
        self.ppm.set_state(f.to(self.ppm.device))

    def get_state(self):
        return self.ppm.get_state()

    # ---- the halo exchange ----
    def pack(self, axis):
        for side in (0, 1):
            if (axis, side) in self.send:
                self.ppm.pack_halo(axis, side, self.send[(axis, side)])
                self.halo_bytes += self.send[(axis, side)].numel() * 4

    def _dist_exchange(self, axis):
        # NCCL enqueues on its own stream, ordered after / before the current torch stream = the library's stream
        with torch.cuda.stream(self.ppm.stream):
            exchange_layers(self.decomp, self.rank, axis, {s: self.send.get((axis, s)) for s in (0, 1)},
                            {s: self.recv.get((axis, s)) for s in (0, 1)}, self.group)

    def exchange(self, axis):
        if self.decomp.procs[axis] > 1:
            self.pack(axis)
            self._exchange(axis)

    # ---- the step (ppm_step's three sweeps, an exchange before each; S10 fused into the last) ----
    def step(self, dt, order=0):
        for s, axis in enumerate(ORDERS[order]):
            self.exchange(axis)
            (self.ppm.sweep_cfl if s == 2 else self.ppm.sweep)(dt, axis)

    def cfl_dt(self, cfl):
        """min over the sub-domains of cfl dx / max(|u| + c): the dt of the undivided grid (a 4- / 8-byte all-reduce)"""
        dt = self.ppm.cfl_dt(cfl)
        if self.decomp.size > 1 and self._exchange == self._dist_exchange:
            import torch.distributed as dist
            t = torch.tensor([dt], dtype=torch.float64, device=self.ppm.device if dist.get_backend(self.group) == "nccl" else "cpu")
            dist.all_reduce(t, op=dist.ReduceOp.MIN, group=self.group)
            dt = float(t.item())
        return dt

    def reduce_conserved(self):
        """sum over the sub-domains of the six conserved totals (a 48-byte all-reduce)"""
        c = self.ppm.reduce_conserved()
        if self.decomp.size > 1 and self._exchange == self._dist_exchange:
            import torch.distributed as dist
            t = torch.tensor(c, dtype=torch.float64, device=self.ppm.device if dist.get_backend(self.group) == "nccl" else "cpu")
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            c = t.cpu().numpy()
        return c

    def close(self):
        self.ppm.close()


class LocalCluster:
    """All sub-domains of a decomposition in ONE process on ONE device: the exchange is a device copy from the sender's packed
    layer into the receiver's halo buffer, everything on one stream, so no kernel ever waits for another.  Same calls as a
    single grid; used by the GPU tests (decomposed == undivided, bit for bit) and to run a decomposed grid without NCCL."""

    def __init__(self, decomp, dx, gamma, grav=None, rho_floor=1e-10, p_floor=1e-10, device="cuda:0"):
        self.decomp = decomp
        self.parts = [DecomposedPPM(decomp, r, dx, gamma, grav, rho_floor, p_floor, device, exchange=lambda axis: None)
                      for r in range(decomp.size)]

    def set_state(self, fields):
        for p in self.parts:
            p.set_state_from_global(fields)

    def get_state(self):
        n = self.decomp.n
        out = torch.empty((15, n[2], n[1], n[0]), dtype=torch.float32, device=self.parts[0].ppm.device)
        for p in self.parts:
            bx, by, bz = p.box()
            out[:, bz, by, bx] = p.get_state()
        return out

    def exchange(self, axis):
        if self.decomp.procs[axis] == 1:
            return
        for p in self.parts:
            p.pack(axis)
        for p in self.parts:
            for side in (0, 1):
                q = self.decomp.neighbour(p.rank, axis, side)
                if q is not None:
                    self.parts[q].recv[(axis, 1 - side)].copy_(p.send[(axis, side)])

    def step(self, dt, order=0):
        for s, axis in enumerate(ORDERS[order]):
            self.exchange(axis)
            for p in self.parts:
                (p.ppm.sweep_cfl if s == 2 else p.ppm.sweep)(dt, axis)

    def cfl_dt(self, cfl):
        return min(p.ppm.cfl_dt(cfl) for p in self.parts)

    def reduce_conserved(self):
        return np.sum([p.ppm.reduce_conserved() for p in self.parts], axis=0)

    def close(self):
        for p in self.parts:
            p.close()
