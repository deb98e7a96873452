"""Plumbing of the domain-decomposed operator: device buffers, streams and the exchange of the
half-spinor faces between sub-lattices.  Every arithmetic step runs in libwd.so (wd_dd_pack, wd_apply on a local
handle, wd_dd_exterior); this module only allocates torch tensors, orders the calls and moves buffers:

  * `LocalOperator`          one sub-lattice: a wd_create_local handle and its eight face buffers per decomposed
                             direction (send / receive, minus / plus);
  * `exchange_on_one_device` all sub-lattices live on ONE GPU (tests; one GPU is all a run has here): a receive
                             buffer is filled by a device copy of the neighbour's send buffer;
  * `exchange_distributed`   one sub-lattice per rank: torch.distributed point-to-point (NCCL over NVLink; gloo on
                             the CPU in the host-logic tests), issued on a communication stream so that it overlaps
                             with the interior kernel (Alg. 3 "hides communication behind computation").

Who gets what (Alg. 3): send_minus[mu] (lambda on my LOW face) goes to the rank in direction -mu and
is ITS recv_from_plus[mu]; send_plus[mu] (chi on my HIGH face) goes to the rank in direction +mu as ITS
recv_from_minus[mu].
"""
from __future__ import annotations

import numpy as np

from . import (WD_OPT_DEVICE_PACK, wd_apply, wd_build_clover, wd_create, wd_create_local, wd_dd_exterior,
               wd_dd_face_bytes, wd_dd_pack, wd_destroy, wd_get_clover, wd_load_clover, wd_load_gauge, wd_set_option,
               wd_set_stream, wd_spinor_bytes)
from .decomp import Decomposition


def local_clover(decomp: Decomposition, rank: int, m0: float, csw: float, U_extended: np.ndarray) -> np.ndarray:
    """S of the local sites from the links of the local lattice EXTENDED by one site in every decomposed direction
    (the clover leaves of eq. 1.12 reach x +- mu +- nu): built on the device on the extended block as a small periodic
    lattice (only its outermost layer sees the wrong wrap) and cut back to the local sites."""
    ext = decomp.extended_dims(1)
    h = wd_create(*ext, m0, csw)
    try:
        wd_load_gauge(h, U_extended)
        wd_build_clover(h)
        C = np.empty((int(np.prod(ext)), 42, 2))
        wd_get_clover(h, C)
    finally:
        wd_destroy(h)
    return np.ascontiguousarray(C[decomp.interior_of_extended(1)])


class LocalOperator:
    def __init__(self, torch, decomp: Decomposition, rank: int, m0: float, csw: float, U_local, C_local=None,
                 device_pack: bool = True):
        self.torch, self.decomp, self.rank = torch, decomp, rank
        self.h = wd_create_local(decomp.global_dims, decomp.grid, decomp.coords(rank), m0, csw)
        self.stream = torch.cuda.current_stream()
        wd_set_stream(self.h, self.stream.cuda_stream)
        wd_set_option(self.h, WD_OPT_DEVICE_PACK, 1 if device_pack else 0)
        wd_load_gauge(self.h, U_local)
        if C_local is not None:
            wd_load_clover(self.h, C_local)
        self.buf = {}  # (mu, name) -> tensor; allocated for nrhs on first use

    def _buffers(self, nrhs: int):
        if self.buf.get("nrhs") != nrhs:
            self.buf = {"nrhs": nrhs}
            for mu in self.decomp.decomposed:
                n = wd_dd_face_bytes(self.h, mu, nrhs) // 8
                for name in ("send_minus", "send_plus", "recv_from_plus", "recv_from_minus"):
                    self.buf[(mu, name)] = self.torch.empty(n, dtype=self.torch.float64, device="cuda")
        return self.buf

    def spinor(self, nrhs: int = 1):
        return self.torch.empty(wd_spinor_bytes(self.h, nrhs) // 8, dtype=self.torch.float64, device="cuda")

    def pack(self, din, nrhs: int = 1):
        b = self._buffers(nrhs)
        for mu in self.decomp.decomposed:
            wd_dd_pack(self.h, din, nrhs, mu, b[(mu, "send_minus")], b[(mu, "send_plus")])

    def interior(self, dout, din, nrhs: int = 1):
        wd_apply(self.h, dout, din, nrhs)

    def exterior(self, dout, nrhs: int = 1):
        b = self._buffers(nrhs)
        for mu in self.decomp.decomposed:
            wd_dd_exterior(self.h, dout, nrhs, mu, b[(mu, "recv_from_plus")], b[(mu, "recv_from_minus")])

    def close(self):
        if self.h:
            wd_destroy(self.h)
            self.h = None


def exchange_on_one_device(ops: list) -> None:
    """All sub-lattices on one device, same stream: a receive buffer is a copy of the neighbour's send buffer."""
    d = ops[0].decomp
    for r, op in enumerate(ops):
        for mu in d.decomposed:
            op.buf[(mu, "recv_from_plus")].copy_(ops[d.neighbour(r, mu, +1)].buf[(mu, "send_minus")])
            op.buf[(mu, "recv_from_minus")].copy_(ops[d.neighbour(r, mu, -1)].buf[(mu, "send_plus")])


def p2p_plan(decomp: Decomposition, rank: int) -> list:
    """The point-to-point operations of one exchange for `rank`, in the order every rank posts them:
    (kind, buffer name, mu, peer rank, tag).  Same relative order on both ends of every pair, so that untagged
    transports (NCCL) match sends and receives correctly even when both neighbours are the same rank."""
    plan = []
    for mu in decomp.decomposed:
        plan.append(("send", "send_minus", mu, decomp.neighbour(rank, mu, -1), 2 * mu))
        plan.append(("send", "send_plus", mu, decomp.neighbour(rank, mu, +1), 2 * mu + 1))
        plan.append(("recv", "recv_from_plus", mu, decomp.neighbour(rank, mu, +1), 2 * mu))
        plan.append(("recv", "recv_from_minus", mu, decomp.neighbour(rank, mu, -1), 2 * mu + 1))
    return plan


def exchange_distributed(dist, decomp: Decomposition, rank: int, buffers: dict) -> list:
    """Posts one exchange with torch.distributed; returns the work handles (wait on them before the exterior step)."""
    ops = []
    for kind, name, mu, peer, tag in p2p_plan(decomp, rank):
        fn = dist.isend if kind == "send" else dist.irecv
        ops.append(dist.P2POp(fn, buffers[(mu, name)], peer, tag=tag))
    return dist.batch_isend_irecv(ops) if ops else []


class DistributedOperator:
    """One rank of the decomposed operator: out = D in on the global lattice, this rank's part."""

    def __init__(self, torch, dist, local: LocalOperator):
        self.torch, self.dist, self.local = torch, dist, local
        self.comm = torch.cuda.Stream()
        self.packed = torch.cuda.Event()

    def apply(self, dout, din, nrhs: int = 1):
        lo, torch = self.local, self.torch
        lo.pack(din, nrhs)
        self.packed.record(lo.stream)
        with torch.cuda.stream(self.comm):  # the exchange runs beside the interior kernel
            self.comm.wait_event(self.packed)
            reqs = exchange_distributed(self.dist, lo.decomp, lo.rank, lo.buf)
        lo.interior(dout, din, nrhs)
        with torch.cuda.stream(self.comm):
            for r in reqs:
                r.wait()
        lo.stream.wait_stream(self.comm)
        lo.exterior(dout, nrhs)


class EmulatedDecomposition:
    """Every sub-lattice of a decomposition on ONE device (how the decomposed path is proven with one GPU): the
    faces are exchanged through device buffers.  Host canonical global fields in, host canonical global field out."""

    def __init__(self, torch, global_dims, grid, m0: float, csw: float, U_global: np.ndarray, C_global=None):
        self.torch = torch
        self.decomp = Decomposition(tuple(global_dims), tuple(grid))
        self.ops = []
        for r in range(self.decomp.world_size):
            Ul = self.decomp.extract(U_global, r)
            if C_global is not None:
                Cl = self.decomp.extract(C_global, r)
            elif csw != 0.0:
                Cl = local_clover(self.decomp, r, m0, csw, self.decomp.extract(U_global, r, halo=1))
            else:
                Cl = None
            self.ops.append(LocalOperator(torch, self.decomp, r, m0, csw, Ul, Cl))

    def apply(self, psi_global: np.ndarray, nrhs: int = 1) -> np.ndarray:
        from . import wd_pack_spinor, wd_synchronize, wd_unpack_spinor

        d = self.decomp
        psi_global = np.ascontiguousarray(psi_global, dtype=np.float64).reshape(nrhs, -1, 12, 2)
        dins, douts = [], []
        for r, op in enumerate(self.ops):
            loc = np.stack([d.extract(psi_global[k], r) for k in range(nrhs)])
            din, dout = op.spinor(nrhs), op.spinor(nrhs)
            dout.fill_(float("nan"))
            wd_pack_spinor(op.h, din, loc, nrhs)
            dins.append(din)
            douts.append(dout)
        for op, din in zip(self.ops, dins):
            op.pack(din, nrhs)
        exchange_on_one_device(self.ops)
        for op, din, dout in zip(self.ops, dins, douts):
            op.interior(dout, din, nrhs)
            op.exterior(dout, nrhs)
        out = np.empty_like(psi_global)
        for r, (op, dout) in enumerate(zip(self.ops, douts)):
            wd_synchronize(op.h)
            loc = np.empty((nrhs, int(np.prod(d.local_dims)), 12, 2))
            wd_unpack_spinor(op.h, loc, dout, nrhs)
            for k in range(nrhs):
                d.insert(out[k], r, loc[k])
        return out

    def close(self):
        for op in self.ops:
            op.close()
        self.ops = []
