"""Element-partitioned runs of the hot path (the paper ran on 3 and 16 GPUs).

One process per GPU, one partition per process.  A rank advances its owned elements with the same kernels as a single-GPU
run; what crosses ranks are two kinds of face data of the partition-boundary faces, every Runge-Kutta stage:
    field 0  face traces of the state being evaluated (9 n^2 doubles per face)   before the element kernel
    field 1  own-side viscous face fluxes (7 n^2 doubles per face, diffusion)     between the element and the face kernel
and one max-allreduce of a double for the CFL wave speed.  The library packs / unpacks the faces into contiguous device
buffers (chorus_halo_pack / chorus_halo_unpack); this module moves the buffers:
    * `DistributedChorus`: torch.distributed all_to_all_single on the packed buffers (NCCL over NVLink / NVSwitch; every
      peer is equidistant, so one all-to-all per exchange with per-peer split sizes is the natural collective);
    * `EmulatedPartitions`: P partitions in ONE process on one GPU, the exchange done by device copies -- the same pack,
      route and unpack path without a network, used to test that results do not depend on P.
Both only marshal: every arithmetic step runs in the CUDA kernels behind include/chorus.h.
"""
from __future__ import annotations

import numpy as np

from . import inputs as I
from .binding import Chorus


def _face_width(order: int, field: int) -> int:
    return (9 if field == 0 else 7) * order * order


def route_offsets(counts) -> np.ndarray:
    """Start of every peer's group in a buffer grouped by peer: [0, c0, c0+c1, ...]."""
    return np.concatenate([[0], np.cumsum(np.asarray(counts, np.int64))])


class _Part:
    """One partition: its library context, halo lists and device buffers."""

    def __init__(self, part: dict, order: int, phys, diffusion: bool):
        import torch
        self.info = part
        self.g = Chorus(part["mesh"], order, phys)
        self.g.set_owned(part["n_owned"])
        self.g.halo_setup(part["send_elem"], part["send_face"], part["recv_elem"], part["recv_face"])
        self.n_send, self.n_recv = int(part["send_counts"].sum()), int(part["recv_counts"].sum())
        wmax = _face_width(order, 0)
        self.send = torch.empty((max(self.n_send, 1), wmax), dtype=torch.float64, device="cuda")
        self.recv = torch.empty((max(self.n_recv, 1), wmax), dtype=torch.float64, device="cuda")
        self.order, self.diffusion = order, diffusion

    def views(self, field: int):
        w = _face_width(self.order, field)
        s = self.send.view(-1)[: self.n_send * w].view(self.n_send, w)
        r = self.recv.view(-1)[: self.n_recv * w].view(self.n_recv, w)
        return s, r


class _Stepper:
    """The stage sequence shared by both drivers; `exchange(field)` moves the halo of that field for all local partitions."""

    def _parts(self):
        raise NotImplementedError

    def exchange(self, field: int):
        raise NotImplementedError

    def step(self, dt: float, nstages: int = 5):
        parts = self._parts()
        for p in parts:
            p.g.step_begin(dt, nstages)
        for i in range(nstages):
            self.exchange(0)                      # ghosts' traces of the state this stage evaluates
            for p in parts:
                p.g.stage_main(i)
            if self.diffusion:
                self.exchange(1)                  # ghosts' own-side viscous face fluxes
            for p in parts:
                p.g.stage_face(i)


class EmulatedPartitions(_Stepper):
    """P partitions of `mesh` advanced in one process on one GPU; the halo travels by device copies between their buffers."""

    def __init__(self, mesh: dict, order: int, phys, n_parts: int):
        self.order, self.P = order, int(n_parts)
        self.diffusion = bool(phys.flags & I.FLAG_DIFFUSION)
        self.E = int(mesh["n_elem"])
        self.parts = [_Part(p, order, phys, self.diffusion) for p in I.partition_mesh(mesh, self.P)]

    def _parts(self):
        return self.parts

    def set_physics(self, phys):
        self.diffusion = bool(phys.flags & I.FLAG_DIFFUSION)
        for p in self.parts:
            p.g.set_physics(phys)

    def set_state(self, Q: np.ndarray):
        """Q: the GLOBAL state [9][E][n^3]; every partition takes its owned and ghost elements."""
        for p in self.parts:
            p.g.set_state(np.ascontiguousarray(Q[:, p.info["elems"]]))

    def get_state(self) -> np.ndarray:
        out = np.empty((9, self.E, self.order ** 3))
        for p in self.parts:
            q = p.g.get_state()
            n = p.info["n_owned"]
            out[:, p.info["elems"][:n]] = q[:, :n]
        return out

    def exchange(self, field: int):
        for p in self.parts:
            s, _ = p.views(field)
            if p.n_send:
                p.g.halo_pack(field, s)
        for p in self.parts:                      # route: rank p's group for q -> rank q's group from p
            so = route_offsets(p.info["send_counts"])
            s, _ = p.views(field)
            for q, dst in enumerate(self.parts):
                cnt = int(p.info["send_counts"][q])
                if cnt == 0:
                    continue
                ro = route_offsets(dst.info["recv_counts"])
                _, r = dst.views(field)
                r[ro[p.info["rank"]]: ro[p.info["rank"]] + cnt].copy_(s[so[q]: so[q] + cnt])
        for p in self.parts:
            _, r = p.views(field)
            if p.n_recv:
                p.g.halo_unpack(field, r)

    def max_wavespeed(self) -> float:
        return max(p.g.max_wavespeed() for p in self.parts)

    def diagnostics(self) -> dict:
        s = sum(p.g.diagnostics_sums() for p in self.parts)
        return dict(V=float(s[0]), KE=float(s[1] / s[0]), EB=float(s[2] / s[0]))

    def launch_count(self) -> int:
        return sum(p.g.launch_count() for p in self.parts)


class DistributedChorus(_Stepper):
    """This process's partition of `mesh` (rank / world size from torch.distributed, backend nccl)."""

    def __init__(self, mesh: dict, order: int, phys, dist):
        self.dist = dist
        self.rank, self.P = dist.get_rank(), dist.get_world_size()
        self.order = order
        self.diffusion = bool(phys.flags & I.FLAG_DIFFUSION)
        self.E = int(mesh["n_elem"])
        self.part = _Part(I.partition_mesh(mesh, self.P, self.rank), order, phys, self.diffusion)
        self.g = self.part.g

    def _parts(self):
        return [self.part]

    def set_physics(self, phys):
        self.diffusion = bool(phys.flags & I.FLAG_DIFFUSION)
        self.g.set_physics(phys)

    @property
    def elems(self):
        return self.part.info["elems"]

    @property
    def n_owned(self):
        return self.part.info["n_owned"]

    def set_state(self, Q_local: np.ndarray):
        """Q_local: [9][n_local][n^3] for this rank's local elements (self.elems); ghost slots are ignored."""
        self.g.set_state(Q_local)

    def exchange(self, field: int):
        p = self.part
        s, r = p.views(field)
        if p.n_send:
            self.g.halo_pack(field, s)
        self.dist.all_to_all_single(r, s, output_split_sizes=[int(c) for c in p.info["recv_counts"]],
                                    input_split_sizes=[int(c) for c in p.info["send_counts"]])
        if p.n_recv:
            self.g.halo_unpack(field, r)

    def max_wavespeed(self) -> float:
        import torch
        t = torch.tensor([self.g.max_wavespeed()], dtype=torch.float64, device="cuda")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def diagnostics(self) -> dict:
        import torch
        t = torch.from_numpy(self.g.diagnostics_sums()).cuda()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        s = t.cpu().numpy()
        return dict(V=float(s[0]), KE=float(s[1] / s[0]), EB=float(s[2] / s[0]))
