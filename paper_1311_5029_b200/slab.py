"""t-slab decomposition: the plumbing around ok_slab_* (include/ok.h) -- no arithmetic of the method.

The lattice is cut along T into equal slabs (only nearest neighbours in time; off-node
communication only for the outermost boundary surfaces).  This module
  * cuts canonical host arrays (links with their OK_SLAB_LINK_HALO = 2 extra slices, spinors) into slab pieces,
  * and provides the two ok_comm callbacks on top of torch.distributed (NCCL on GPUs, gloo on CPU tensors in the tests):
    the exchange of one boundary time slice with each t-neighbour rank and the all-gather of the per-slab partial sums.
One process per GPU; a process may hold several consecutive slabs.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import binding as B


def slab_ranges(T: int, nslab_total: int):
    """[(t0, Tloc)] of nslab_total equal slabs of a lattice of T time slices."""
    if T % nslab_total:
        raise ValueError(f"T = {T} is not a multiple of {nslab_total} slabs")
    Tloc = T // nslab_total
    return [(s * Tloc, Tloc) for s in range(nslab_total)]


def link_window(U: np.ndarray, dims, t0: int, Tloc: int) -> np.ndarray:
    """Canonical links [V][4][3][3] of the whole lattice -> those of the global slices t0 - 2 .. t0 + Tloc + 1 (mod T)."""
    slice_sites = dims[0] * dims[1] * dims[2]
    T = dims[3]
    ts = [(t0 - B.OK_SLAB_LINK_HALO + k) % T for k in range(Tloc + 2 * B.OK_SLAB_LINK_HALO)]
    Ut = U.reshape(T, slice_sites, 4, 3, 3)
    return np.ascontiguousarray(Ut[ts]).reshape(-1, 4, 3, 3)


def spinor_slab(psi: np.ndarray, dims, t0: int, Tloc: int) -> np.ndarray:
    """Canonical spinor [V][12] -> the slab's own Tloc slices."""
    slice_sites = dims[0] * dims[1] * dims[2]
    return np.ascontiguousarray(psi.reshape(dims[3], slice_sites, 12)[t0:t0 + Tloc]).reshape(-1, 12)


def interior(slab: B.ok_params, vec_ext):
    """The ordinary internal-layout field of the slab's own lattice inside an extended field (a view)."""
    sb = B.ok_slab_slice_bytes(slab)
    return vec_ext[sb:sb + sb * slab.dims[3]]


def halo_views(slab: B.ok_params, vec_ext):
    """(lower halo, first slice, last slice, upper halo) of an extended field (views, bytes)."""
    sb, Tl = B.ok_slab_slice_bytes(slab), slab.dims[3]
    return vec_ext[0:sb], vec_ext[sb:2 * sb], vec_ext[Tl * sb:(Tl + 1) * sb], vec_ext[(Tl + 1) * sb:(Tl + 2) * sb]


class TorchComm:
    """ok_comm over torch.distributed.  The callbacks get raw addresses; they are turned back into views of the torch tensors
    the caller registered (the workspace and the x fields -- every buffer the solver exchanges lives in one of them)."""

    def __init__(self, dist, stream=None, group=None):
        import torch
        self.torch, self.dist, self.group, self.stream = torch, dist, group, stream
        self.rank, self.nranks = dist.get_rank(group), dist.get_world_size(group)
        self.buffers = []
        self._ex = B.EXCHANGE_FN(self._exchange)
        self._ag = B.ALLGATHER_FN(self._allgather)
        self.struct = B.ok_comm(self.rank, self.nranks, self._ex, self._ag, None)
        self.error = None

    def register(self, *tensors):
        """uint8 tensors that contain every address the library may pass to the callbacks."""
        self.buffers.extend(tensors)

    def view(self, addr, nbytes):
        for t in self.buffers:
            off = addr - t.data_ptr()
            if 0 <= off and off + nbytes <= t.numel() * t.element_size():
                return t.view(self.torch.uint8).reshape(-1)[off:off + nbytes]
        raise RuntimeError("ok_comm callback: address outside the registered buffers")

    def exchange_tensors(self, send_lo, send_hi, recv_lo, recv_hi):
        """send_lo -> rank - 1 (arrives in its recv_hi); send_hi -> rank + 1 (arrives in its recv_lo); cyclic."""
        dist, n, r = self.dist, self.nranks, self.rank
        if n == 1:
            recv_hi.copy_(send_lo)
            recv_lo.copy_(send_hi)
            return
        down, up = (r - 1) % n, (r + 1) % n
        ops = [dist.P2POp(dist.isend, send_lo, down, self.group), dist.P2POp(dist.isend, send_hi, up, self.group),
               dist.P2POp(dist.irecv, recv_hi, up, self.group), dist.P2POp(dist.irecv, recv_lo, down, self.group)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()

    def allgather_tensors(self, send, recv):
        """recv[r * n : (r + 1) * n] = rank r's send."""
        if self.nranks == 1:
            recv.copy_(send)
        elif send.is_cuda and self.dist.get_backend(self.group) == "gloo":   # gloo has no all-gather on device tensors: stage on the host
            host = self.torch.empty(recv.numel(), dtype=recv.dtype)
            self.dist.all_gather_into_tensor(host, send.cpu(), group=self.group)
            recv.copy_(host)
        else:
            self.dist.all_gather_into_tensor(recv, send, group=self.group)

    def _on_stream(self):
        import contextlib
        return self.torch.cuda.stream(self.stream) if self.stream is not None else contextlib.nullcontext()

    def _exchange(self, user, send_lo, send_hi, recv_lo, recv_hi, nbytes):
        try:
            with self._on_stream():   # the collectives order themselves against the library's stream
                self.exchange_tensors(self.view(send_lo, nbytes), self.view(send_hi, nbytes), self.view(recv_lo, nbytes),
                                      self.view(recv_hi, nbytes))
            return 0
        except Exception as e:      # an exception must not cross the C boundary
            self.error = e
            return 1

    def _allgather(self, user, send, recv, n):
        try:
            with self._on_stream():
                s = self.view(send, 8 * n).view(self.torch.float64)
                r = self.view(recv, 8 * n * self.nranks).view(self.torch.float64)
                self.allgather_tensors(s, r)
            return 0
        except Exception as e:
            self.error = e
            return 1


class PeerLinks:
    """ok_slab_peers over torch (include/ok.h: ok_slab_set_peers): maps the two t-neighbour processes' workspace and x buffers
    into this process -- CUDA IPC through torch's own tensor sharing, i.e. NVLink peer access when the neighbour sits on another
    GPU -- and provides the barrier callback.  Every rank passes its workspace tensor and the x_ext tensors of its first and
    last slab; keep this object (and the tensors) alive while the peers are set, and delete it before the buffers are freed."""

    def __init__(self, dist, work, x_first, x_last, group=None, stream=None):
        import torch
        from torch.multiprocessing.reductions import reduce_tensor
        self.torch, self.dist, self.group, self.stream = torch, dist, group, stream
        rank, n = dist.get_rank(group), dist.get_world_size(group)
        mine = tuple(reduce_tensor(t) for t in (work, x_first, x_last))      # picklable (rebuild function, IPC handle) pairs
        everyone = [None] * n
        dist.all_gather_object(everyone, mine, group=group)
        opened = lambda h: h[0](*h[1])
        lo, hi = everyone[(rank - 1) % n], everyone[(rank + 1) % n]
        self.lo_work, self.lo_x = opened(lo[0]), opened(lo[2])                # the lower neighbour's LAST slab
        self.hi_work, self.hi_x = opened(hi[0]), opened(hi[1])                # the upper neighbour's FIRST slab
        self.error = None
        self._bar = B.BARRIER_FN(self._barrier)
        self.struct = B.ok_slab_peers(self.lo_work.data_ptr(), self.hi_work.data_ptr(), self.lo_x.data_ptr(), self.hi_x.data_ptr(),
                                      self._bar, None)

    def _barrier(self, user):
        try:   # everything enqueued so far is complete on every rank before anyone goes on
            (self.stream.synchronize() if self.stream is not None else self.torch.cuda.synchronize())
            self.dist.barrier(group=self.group)
            return 0
        except Exception as e:
            self.error = e
            return 1

