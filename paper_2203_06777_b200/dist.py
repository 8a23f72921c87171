"""Time-direction domain decomposition of Dhop over several GPUs.

Plumbing only: every arithmetic step runs in libdwf's kernels (``dwf_dhop_oe/eo`` on a geometry with an open time
boundary, ``dwf_face_pack_t``, ``dwf_face_apply_t``); this module decides who sends which face buffer to whom and
moves the buffers -- ``torch.distributed`` point-to-point operations between ranks (one process per GPU, NCCL),
or plain device copies when a rank is its own neighbour -- on a side stream, while the bulk kernel computes.

The lattice is cut into ``world`` slabs along time (x3; the fifth dimension is never split).  Rank r owns the time
layers ``[r * L3/world, (r+1) * L3/world)``; its lower neighbour is rank r-1, its upper neighbour rank r+1
(periodically).  With a globally antiperiodic time direction the face that crosses the global boundary (rank 0's
lower face, the last rank's upper face) carries the factor -1.
"""
from __future__ import annotations

from . import (ANTIPERIODIC_T, EVEN, ODD, OPEN_T, Geometry, dwf_face_apply_t, dwf_face_bytes, dwf_face_pack_t)


def slab_plan(rank: int, world: int, L3: int, bc_time_global: int):
    """Who my neighbours are, which time layers I own and the sign of my two faces.  Pure host logic."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world")
    if L3 % world or (L3 // world) % 2 or L3 // world < 2:
        raise ValueError("the time extent must split into slabs of an even number (>= 2) of layers")
    l3 = L3 // world
    anti = bc_time_global == ANTIPERIODIC_T
    return {
        "lower": (rank - 1) % world, "upper": (rank + 1) % world,
        "t0": rank * l3, "t1": (rank + 1) * l3, "local_L3": l3,
        "sign_lo": -1.0 if (anti and rank == 0) else 1.0,
        "sign_hi": -1.0 if (anti and rank == world - 1) else 1.0,
    }


def exchange_faces(send_down, send_up, recv_lo, recv_hi, rank: int, world: int, group=None):
    """recv_lo <- the lower neighbour's send_up, recv_hi <- the upper neighbour's send_down.  Works on CUDA tensors
    (NCCL) and on CPU tensors (gloo: the host-side test of the pattern).  world == 1: the rank is its own neighbour."""
    if world == 1:
        recv_lo.copy_(send_up)
        recv_hi.copy_(send_down)
        return
    import torch.distributed as dist
    lower, upper = (rank - 1) % world, (rank + 1) % world
    ops = [dist.P2POp(dist.isend, send_up, upper, group), dist.P2POp(dist.irecv, recv_lo, lower, group),
           dist.P2POp(dist.isend, send_down, lower, group), dist.P2POp(dist.irecv, recv_hi, upper, group)]
    # world == 2: both neighbours are the same peer; messages between two ranks match in the order they are posted, and
    # both sides post (send_up, recv_lo) first: my send_up pairs with the peer's recv_lo (its lower neighbour is me)
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class SlabDhop:
    """One rank's share of a time-decomposed even/odd Dhop.

        op = SlabDhop(global_dims, Ls, precision, bc_time_global, rank, world, device)
        op.load_gauge(U_slab)                      # canonical links of MY time layers, (V4_slab, 4, 3, 3, 2)
        out = op.dhop_oe(f_even)                   # device fields of the slab geometry (op.geometry)

    `exchange` replaces the transport (tests emulate several ranks in one process on one GPU by handing every
    instance a function that reads the other instances' send buffers)."""

    def __init__(self, global_dims, Ls: int, precision: int, bc_time_global: int, rank: int, world: int, device: int = 0,
                 group=None, exchange=None):
        import torch
        self.plan = slab_plan(rank, world, int(global_dims[3]), bc_time_global)
        self.rank, self.world, self.group = rank, world, group
        dims = tuple(int(d) for d in global_dims[:3]) + (self.plan["local_L3"],)
        self.geometry = Geometry(dims, Ls, precision, OPEN_T, device=device)
        self._torch = torch
        nb = dwf_face_bytes(self.geometry.handle)
        dev = f"cuda:{device}"
        mk = lambda: torch.empty(nb // precision, dtype=self.geometry.torch_dtype, device=dev)
        self.send_down, self.send_up, self.recv_lo, self.recv_hi = mk(), mk(), mk(), mk()
        self.comm_stream = torch.cuda.Stream(device=dev)
        self._exchange = exchange

    def close(self):
        self.geometry.close()

    def load_gauge(self, U_slab):
        self.geometry.load_gauge(U_slab)

    # The three phases of a half-Dhop.  A real run calls them back to back (_half); the single-GPU emulation of
    # several ranks in the tests runs each phase for all virtual ranks before the next one.
    def pack(self, f_in, parity_out: int, dagger: bool = False):
        """1. faces of the input (parity 1 - parity_out), on the current stream"""
        torch, g = self._torch, self.geometry
        dwf_face_pack_t(g.handle, f_in, 1 - parity_out, self.send_down, self.send_up, dagger)
        self._packed = torch.cuda.Event()
        self._packed.record(torch.cuda.current_stream(g.device))

    def communicate(self):
        """2. the exchange, on the side stream (so that the bulk kernel issued next overlaps it)"""
        torch = self._torch
        with torch.cuda.stream(self.comm_stream):
            self.comm_stream.wait_event(self._packed)
            if self._exchange is not None:
                self._exchange(self)
            else:
                exchange_faces(self.send_down, self.send_up, self.recv_lo, self.recv_hi, self.rank, self.world, self.group)
            self._arrived = torch.cuda.Event()
            self._arrived.record(self.comm_stream)

    def bulk_and_faces(self, f_in, parity_out: int, dagger: bool = False, out=None):
        """3. the bulk kernel (open time boundary), 4. the two face terms once the buffers have arrived"""
        torch, g = self._torch, self.geometry
        out = g.new_field(parity_out) if out is None else out
        if parity_out == ODD:
            (g.dhop_oe_dag if dagger else g.dhop_oe)(f_in, out)
        else:
            (g.dhop_eo_dag if dagger else g.dhop_eo)(f_in, out)
        torch.cuda.current_stream(g.device).wait_event(self._arrived)
        dwf_face_apply_t(g.handle, self.recv_lo, self.recv_hi, self.plan["sign_lo"], self.plan["sign_hi"], out, parity_out, dagger)
        return out

    def _half(self, f_in, parity_out: int, dagger: bool, out=None):
        self.pack(f_in, parity_out, dagger)
        self.communicate()
        return self.bulk_and_faces(f_in, parity_out, dagger, out)

    def dhop_oe(self, f_even, out=None, dagger: bool = False):
        return self._half(f_even, ODD, dagger, out)

    def dhop_eo(self, f_odd, out=None, dagger: bool = False):
        return self._half(f_odd, EVEN, dagger, out)
