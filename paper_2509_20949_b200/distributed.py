"""Lattice parallelism with one slab per process / GPU (include/smcx.h "Lattice parallelism").

Every rank holds one ``Domain`` (``smcx_domain_t``): slab ``rank`` of the lattice cut into ``world_size`` slabs along z.
The kernels, the message plan (which bytes of the species storage travel when) and the partial reductions all live
behind the C ABI; this module only moves the messages -- ``torch.distributed`` point-to-point operations on views of
the workspace tensor (NCCL over NVLink between GPUs: plumbing, as for the single-GPU path) -- and sums the partial
results.  With ``overlap`` a colour pass is launched as its boundary row first; the row's layers are in flight on a
side stream while the other rows of the pass run (computation-communication overlap).

``exchange`` is the whole transport.  The same function moves the messages between slabs that live in one process
(``LocalWorld``, used by the one-GPU tests), so the ordering logic is exercised without a second GPU.
"""
from __future__ import annotations

import numpy as np

from . import binding as _b


class LocalWorld:
    """Stand-in for a process group whose ranks all live in this process: a message is a tensor copy."""

    def __init__(self, n):
        self.n = int(n)
        self.mail = {}

    def post(self, src_rank, msg, view):
        peer, tag, _, nbytes = msg
        if nbytes:
            self.mail[(src_rank, peer, tag)] = view

    def deliver(self, dst_rank, msg, view):
        peer, tag, _, nbytes = msg
        if nbytes:
            view.copy_(self.mail.pop((peer, dst_rank, tag)))


def exchange(dist, rank, storage_view, send, recv, group=None):
    """Post the messages of one phase with torch.distributed: the receive first, then the send; returns the work
    handles.  A message is (peer, tag, offset, bytes); bytes == 0 means none.  A phase has at most one outgoing and
    one incoming message per slab (reading S11), so a send can only match the peer's one receive -- also between two
    slabs of a periodic lattice, which are each other's lower and upper neighbour."""
    ops = []
    for kind, msg in (("recv", recv), ("send", send)):
        peer, _tag, off, nbytes = msg
        if not nbytes:
            continue
        view = storage_view[off: off + nbytes]
        ops.append(dist.P2POp(dist.irecv if kind == "recv" else dist.isend, view, peer, group))
    return dist.batch_isend_irecv(ops) if ops else []


class SlabRank:
    """One slab of a distributed lattice.  ``dist`` is ``torch.distributed`` (initialised by the caller, e.g. under
    torchrun with the NCCL backend) or None when ``world`` is a LocalWorld shared by the slabs of one process."""

    def __init__(self, rank, world_size, dist=None, world=None, overlap=True, domain=None, **lattice_kw):
        import torch

        self.torch = torch
        self.rank, self.world_size = int(rank), int(world_size)
        self.dist, self.world = dist, world
        self.overlap = bool(overlap)
        # `domain`: an object with Domain's stepping calls and a `_storage_view` tensor (the host-side tests pass a
        # stand-in whose storage is a CPU tensor, to run this driver over gloo); by default the slab on the GPU
        self.domain = domain if domain is not None else _b.Domain(self.world_size, self.rank, **lattice_kw)
        self.compute = getattr(self.domain, "_stream", None)
        self.side = None
        if self.compute is not None:
            with torch.cuda.device(self.domain.device):
                self.side = torch.cuda.Stream(device=self.domain.device)
        self._kw = {k: lattice_kw[k] for k in ("lattice", "dims", "n_species", "n_shells", "epi", "accept", "seed") if k in lattice_kw}
        self._kw["link_cell"] = lattice_kw.get("link_cell", 4)
        self.message_bytes = 0

    # -- transport ------------------------------------------------------------------------------------------
    def _start(self, send, recv):
        """Begin moving one phase's messages once the work enqueued so far on the compute stream is done."""
        self.message_bytes += send[3]
        if self.dist is None:
            self.world.post(self.rank, send, self.domain.storage_view(send))
            return (send, recv)
        if self.side is None:                      # host stand-in: no streams to order
            return exchange(self.dist, self.rank, self.domain._storage_view, send, recv)
        self.side.wait_stream(self.compute)
        with self.torch.cuda.stream(self.side):
            return exchange(self.dist, self.rank, self.domain._storage_view, send, recv)

    def _finish(self, pending):
        """The compute stream waits for the phase's incoming and outgoing messages."""
        if self.dist is None:
            _send, recv = pending
            self.world.deliver(self.rank, recv, self.domain.storage_view(recv))
            return
        for work in pending:
            work.wait()            # NCCL: orders the current (compute) stream after the transfer
        if getattr(self, "_side_busy", False):
            self.compute.wait_stream(self.side)      # ... and after the boundary row itself
            self._side_busy = False

    # -- one sweep, in the three steps a LocalWorld needs (post everything, then deliver) --------------------
    def sweep_begin(self):
        return self._start(*self.domain.begin_sweep())

    def pass_begin(self, colour):
        send, recv = self.domain.pass_messages(colour)
        if self.overlap and self.side is not None and self.dist is not None:
            # boundary row on the side stream, the other rows on the compute stream, at the same time; the message
            # leaves from the side stream as soon as the boundary row is done
            self.domain.run_pass_split(colour, self.side)
            self.message_bytes += send[3]
            with self.torch.cuda.stream(self.side):
                pending = exchange(self.dist, self.rank, self.domain._storage_view, send, recv)
            self._side_busy = True
        elif self.overlap:
            self.domain.run_pass(colour, 1)          # the boundary row, whose layers the message carries
            pending = self._start(send, recv)
            self.domain.run_pass(colour, 2)          # the other rows run while the message is in flight
        else:
            self.domain.run_pass(colour, 0)
            pending = self._start(send, recv)
        return pending

    def phase_end(self, pending):
        self._finish(pending)

    def sweep_end(self):
        self.domain.end_sweep()

    def sweep(self, n=1):
        """n sweeps when every rank is its own process (torch.distributed)."""
        assert self.dist is not None, "slabs that share a process are stepped by run_local()"
        for _ in range(int(n)):
            self.phase_end(self.sweep_begin())
            for colour in range(8):
                self.phase_end(self.pass_begin(colour))
            self.sweep_end()

    # -- reductions over the slabs ----------------------------------------------------------------------------
    def _allreduce_i64(self, a):
        if self.dist is None:
            return a
        t = self.torch.from_numpy(np.ascontiguousarray(a, dtype=np.int64)).to(self.domain.device)
        self.dist.all_reduce(t)
        return t.cpu().numpy()

    def running_energy(self) -> int:
        return int(self._allreduce_i64(np.array([self.domain.running_energy()]))[0])

    def energy_trace(self, first=0, count=None):
        return self._allreduce_i64(self.domain.energy_trace(first, count))

    def pair_counts(self):
        return self._allreduce_i64(self.domain.pair_counts())

    def sro(self):
        return _b.sro_from_counts(self.pair_counts(), **self._kw)

    def stats(self):
        s, t, a = self.domain.stats()
        tot = self._allreduce_i64(np.array([t, a]))
        return s, int(tot[0]), int(tot[1])

    def close(self):
        self.domain.close()


class ConnectedSlabRank(SlabRank):
    """One slab per process with NO host code in the data path (include/smcx.h, "Connected slabs"): the ranks exchange
    CUDA IPC handles of their slabs once (`dist.all_gather_object`), map their neighbours' storage, and from then on
    `sweep(n)` is one C call that enqueues n whole sweeps -- ghost layers are written by the sweep kernels straight into
    the neighbour's memory (peer stores over NVLink between GPUs of a node) and signalled through device flags.
    torch.distributed carries the handles and the partial reductions only.  All ranks must share a node."""

    def __init__(self, rank, world_size, dist, **lattice_kw):
        import torch

        self.torch = torch
        self.rank, self.world_size = int(rank), int(world_size)
        self.dist, self.world, self.overlap = dist, None, True
        self.domain = _b.Domain(self.world_size, self.rank, library_workspace=True, **lattice_kw)
        self.compute, self.side = self.domain._stream, None
        self._kw = {k: lattice_kw[k] for k in ("lattice", "dims", "n_species", "n_shells", "epi", "accept", "seed") if k in lattice_kw}
        self._kw["link_cell"] = lattice_kw.get("link_cell", 4)
        self.message_bytes = 0
        handles = [None] * self.world_size
        dist.all_gather_object(handles, self.domain.ipc_export())
        self.domain.ipc_connect(handles[(self.rank - 1) % self.world_size], handles[(self.rank + 1) % self.world_size])
        dist.barrier()                               # every slab connected (flags zeroed) before any slab sweeps

    def sweep(self, n=1):
        self.domain.sweep_connected(int(n))

    def close(self):
        self.domain.synchronize()
        self.dist.barrier()                          # nobody unmaps a neighbour that is still being written to
        self.domain.close()


def run_local(slabs, n=1):
    """n sweeps of slabs that share a process and a LocalWorld: every phase is posted by all slabs, then delivered."""
    torch = slabs[0].torch
    for _ in range(int(n)):
        for begin in [lambda s: s.sweep_begin()] + [(lambda s, c=c: s.pass_begin(c)) for c in range(8)]:
            pend = [begin(s) for s in slabs]
            torch.cuda.synchronize()          # slabs of one process share a device in the tests: plain ordering
            for s, p in zip(slabs, pend):
                s.phase_end(p)
            torch.cuda.synchronize()
        for s in slabs:
            s.sweep_end()
