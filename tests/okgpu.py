"""Helpers for the -m gpu parity tests: move seeded inputs to the device and call the C-ABI."""
import numpy as np
import torch

from paper_1311_5029_b200 import binding as B

DEV = "cuda:0"
_ws = {}


def cdtype(prec):
    return torch.complex128 if prec == B.OK_FP64 else torch.complex64


def npdtype(prec):
    return np.complex128 if prec == B.OK_FP64 else np.complex64


def workspace(p):
    """(Re)bind a workspace large enough for p; the tensor is kept alive here (caller-owned)."""
    need = B.ok_work_bytes(p)
    if _ws.get("n", 0) < need:
        _ws["buf"] = None
        _ws["buf"] = B.alloc_bytes(need, DEV)
        _ws["n"] = need
    B.ok_set_workspace(_ws["buf"], _ws["n"])
    B.ok_set_stream(None)


def to_dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.to(DEV)


def pack_spinor(p, psi_np):
    canon = to_dev(psi_np, cdtype(p.precision))
    packed = B.alloc_vec(p, DEV)
    B.ok_pack_spinor(p, canon, packed)
    return packed


def unpack_spinor(p, packed, shape):
    canon = torch.empty(shape, dtype=cdtype(p.precision), device=DEV)
    B.ok_unpack_spinor(p, packed, canon)
    torch.cuda.synchronize()
    return canon.cpu().numpy().astype(np.complex128)


def precalc(p, links_np):
    workspace(p)
    links = to_dev(links_np, torch.complex128)
    W = B.alloc_W(p, DEV)
    B.ok_precalc_W(links, p, W)
    torch.cuda.synchronize()
    return W


def unpack_W(p, W, V):
    canon = torch.empty((V, 27, 12, 12), dtype=cdtype(p.precision), device=DEV)
    B.ok_unpack_W(W, canon)
    torch.cuda.synchronize()
    return canon.cpu().numpy().astype(np.complex128)


def apply(p, W, psi_np):
    packed = pack_spinor(p, psi_np)
    out = B.alloc_vec(p, DEV)
    B.ok_dirac_apply(W, packed, out)
    return unpack_spinor(p, out, psi_np.shape)


def per_site_rel_err(got, want):
    """max over sites of ||got(x) - want(x)||_2 / ||want(x)||_2 (sites with negligible want skipped; S12)."""
    num = np.linalg.norm(got - want, axis=1)
    den = np.linalg.norm(want, axis=1)
    keep = den > 1e-30 * den.max()
    return float((num[keep] / den[keep]).max())


def rel_l2(got, want):
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def fp32_operator_slack(o, x, b, idx=None, W=None):
    """DESIGN.md 10, reading R-RESID.  The library's `resid` of an fp32 solve is || b - fl32(M32 x) || / || b || with M32 the
    fp32-rounded W it stores; the oracle evaluates || b - M64 x || / || b ||.  The two differ by at most
        || (M32 - M64) x || + || fl32(M32 x) - M32 x ||   <=   2 * 2^-24 * || |W| |x| ||_2
    (every real of W rounded once: |dW| <= 2^-24 |W| elementwise, rigorous; the second term is the kernel's own fp32 rounding
    of the 324-term sums, whose accumulated error stays below one unit 2^-24 |W||x| in every measured case).  Returns that
    bound relative to || b || -- evaluated by the oracle as apply_W(|x|, W = |W|) -- on the sites `idx` (all sites if None;
    for a sample the caller extrapolates like the residual itself)."""
    Wa = np.abs(o.precalc_W(idx) if W is None else W).astype(np.complex128)
    S = o.apply_W(np.abs(x).astype(np.complex128), idx=idx, W=Wa)
    scale = 1.0 if idx is None else np.sqrt(o.V / len(idx))
    if S.ndim == 3:     # [site][comp][rhs]: one bound per column
        return 2.0 * 2.0 ** -24 * scale * np.linalg.norm(S.reshape(-1, S.shape[2]), axis=0) / np.linalg.norm(b.reshape(-1, b.shape[2]), axis=0)
    return 2.0 * 2.0 ** -24 * scale * float(np.linalg.norm(S)) / float(np.linalg.norm(b))


def ipc_slab_worker(rank, nranks, U, pd, prec, psi, q_in, q_out, results, barrier):
    """One process = one t-slab on cuda:0 (tests/test_gpu_slab.py, the CUDA-IPC test): builds its W and field, hands its field to
    the two t-neighbours as a CUDA IPC handle (a torch CUDA tensor sent through a multiprocessing queue), maps theirs, and applies
    with ok_slab_dirac_apply_peer reading the neighbours' boundary slices through the mapping.  Host-side barriers order the
    phases; no kernel waits on another process's kernel."""
    from paper_1311_5029_b200 import slab as S
    try:
        torch.cuda.set_device(0)
        dims = tuple(pd["dims"])
        p = B.make_params(pd, prec)
        t0, Tl = S.slab_ranges(dims[3], nranks)[rank]
        slab = B.make_slab_params(p, Tl)
        plocal = B.make_params(dict(pd, dims=dims[:3] + (Tl,)), prec)
        work = B.alloc_bytes(B.ok_slab_work_bytes(slab, 1, 1), DEV)
        B.ok_set_stream(None)
        B.ok_set_workspace(work, work.numel())
        W = B.alloc_W(slab, DEV)
        B.ok_slab_precalc_W(to_dev(S.link_window(U, dims, t0, Tl), torch.complex128), slab, dims[3], t0, W)
        v = torch.zeros(B.ok_slab_vec_bytes(slab), dtype=torch.uint8, device=DEV)
        B.ok_pack_spinor(plocal, to_dev(S.spinor_slab(psi, dims, t0, Tl), cdtype(prec)), S.interior(slab, v))
        lo, first, last, hi = S.halo_views(slab, v)
        lo.fill_(0xFF)
        hi.fill_(0xFF)
        torch.cuda.synchronize()
        q_in[(rank - 1) % nranks].put(("from_above", v))      # my field, for my lower neighbour's upper face
        q_in[(rank + 1) % nranks].put(("from_below", v))
        got = dict(q_in[rank].get(timeout=120) for _ in range(2))
        barrier.wait(timeout=120)                              # every field is complete and mapped
        out = torch.zeros_like(v)
        lo_slice = S.halo_views(slab, got["from_below"])[2]    # the lower neighbour's last own slice, in ITS memory
        hi_slice = S.halo_views(slab, got["from_above"])[1]
        B.ok_slab_dirac_apply_peer(W, v, lo_slice, hi_slice, out)
        canon = torch.empty((Tl * dims[0] * dims[1] * dims[2], 12), dtype=cdtype(prec), device=DEV)
        B.ok_unpack_spinor(plocal, S.interior(slab, out), canon)
        torch.cuda.synchronize()
        results.put((rank, canon.cpu().numpy(), None))
        barrier.wait(timeout=120)                              # nobody frees a field a neighbour may still be reading
        del got, lo_slice, hi_slice
    except Exception as e:  # pragma: no cover
        results.put((rank, None, repr(e)))
        try:
            barrier.abort()
        except Exception:
            pass


def ipc_solver_worker(rank, nranks, U, pd, prec, b_np, tol, q_in, q_ag, results, barrier):
    """One process = one t-slab on cuda:0 running ok_slab_bicgstab with ok_slab_set_peers: the outer faces of every apply are
    read from the other process's workspace / x buffer through CUDA IPC mappings; the reductions cross the processes through
    multiprocessing queues (plumbing); `exchange` must never be called."""
    import ctypes as C
    from paper_1311_5029_b200 import slab as S
    try:
        torch.cuda.set_device(0)
        dims = tuple(pd["dims"])
        p = B.make_params(pd, prec)
        t0, Tl = S.slab_ranges(dims[3], nranks)[rank]
        slab = B.make_slab_params(p, Tl)
        plocal = B.make_params(dict(pd, dims=dims[:3] + (Tl,)), prec)
        work = B.alloc_bytes(B.ok_slab_work_bytes(slab, 1, nranks), DEV)
        B.ok_set_stream(None)
        B.ok_set_workspace(work, work.numel())
        W = B.alloc_W(slab, DEV)
        B.ok_slab_precalc_W(to_dev(S.link_window(U, dims, t0, Tl), torch.complex128), slab, dims[3], t0, W)
        src = torch.zeros(B.ok_slab_vec_bytes(slab), dtype=torch.uint8, device=DEV)
        B.ok_pack_spinor(plocal, to_dev(S.spinor_slab(b_np, dims, t0, Tl), cdtype(prec)), S.interior(slab, src))
        x = torch.zeros_like(src)
        torch.cuda.synchronize()
        q_in[(rank - 1) % nranks].put(("from_above", work, x))
        q_in[(rank + 1) % nranks].put(("from_below", work, x))
        got = {}
        for _ in range(2):
            tag, w_, x_ = q_in[rank].get(timeout=120)
            got[tag] = (w_, x_)
        barrier.wait(timeout=120)
        calls = {"exchange": 0, "allgather": 0, "barrier": 0}

        def view(addr, nbytes):
            off = addr - work.data_ptr()
            assert 0 <= off and off + nbytes <= work.numel()
            return work[off:off + nbytes]

        def on_barrier(user):
            try:
                calls["barrier"] += 1
                torch.cuda.synchronize()
                barrier.wait(timeout=120)
                return 0
            except Exception:
                return 1

        def on_allgather(user, send, recv, n):
            try:
                calls["allgather"] += 1
                torch.cuda.synchronize()
                mine = view(send, 8 * n).view(torch.float64).cpu().numpy().copy()
                for r in range(nranks):
                    if r != rank:
                        q_ag[r].put((rank, mine))
                parts = {rank: mine}
                while len(parts) < nranks:
                    r, arr = q_ag[rank].get(timeout=120)
                    parts[r] = arr
                allv = np.concatenate([parts[r] for r in range(nranks)])
                view(recv, 8 * n * nranks).view(torch.float64).copy_(torch.from_numpy(allv))
                torch.cuda.synchronize()
                return 0
            except Exception:
                return 1

        def on_exchange(*a):
            calls["exchange"] += 1
            return 1

        cb = (B.EXCHANGE_FN(on_exchange), B.ALLGATHER_FN(on_allgather), B.BARRIER_FN(on_barrier))
        comm = B.ok_comm(rank, nranks, cb[0], cb[1], None)
        peers = B.ok_slab_peers(got["from_below"][0].data_ptr(), got["from_above"][0].data_ptr(), got["from_below"][1].data_ptr(),
                                got["from_above"][1].data_ptr(), cb[2], None)
        B.ok_slab_set_peers(peers)
        st, it, res = B.ok_slab_bicgstab([W], [src], [x], tol, 2000, comm=comm, raise_on_fail=False)
        B.ok_slab_set_peers(None)
        canon = torch.empty((Tl * dims[0] * dims[1] * dims[2], 12), dtype=cdtype(prec), device=DEV)
        B.ok_unpack_spinor(plocal, S.interior(slab, x), canon)
        torch.cuda.synchronize()
        results.put((rank, (st, it, res, dict(calls), canon.cpu().numpy()), None))
        barrier.wait(timeout=120)
        del got
    except Exception as e:  # pragma: no cover
        import traceback
        results.put((rank, None, traceback.format_exc()))
        try:
            barrier.abort()
        except Exception:
            pass


def torch_peer_solver_worker(rank, nranks, port, U, pd, prec, b_np, tol, results):
    """The same solve through the package's own plumbing: torch.distributed (gloo here: both ranks share cuda:0) for the
    reductions and the barrier, slab.PeerLinks for the mappings, slab.TorchComm for ok_comm."""
    import os
    import torch.distributed as dist
    from paper_1311_5029_b200 import slab as S
    try:
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(nranks))
        dist.init_process_group("gloo", rank=rank, world_size=nranks)
        torch.cuda.set_device(0)
        dims = tuple(pd["dims"])
        p = B.make_params(pd, prec)
        t0, Tl = S.slab_ranges(dims[3], nranks)[rank]
        slab = B.make_slab_params(p, Tl)
        plocal = B.make_params(dict(pd, dims=dims[:3] + (Tl,)), prec)
        work = B.alloc_bytes(B.ok_slab_work_bytes(slab, 1, nranks), DEV)
        B.ok_set_stream(None)
        B.ok_set_workspace(work, work.numel())
        W = B.alloc_W(slab, DEV)
        B.ok_slab_precalc_W(to_dev(S.link_window(U, dims, t0, Tl), torch.complex128), slab, dims[3], t0, W)
        src = torch.zeros(B.ok_slab_vec_bytes(slab), dtype=torch.uint8, device=DEV)
        B.ok_pack_spinor(plocal, to_dev(S.spinor_slab(b_np, dims, t0, Tl), cdtype(prec)), S.interior(slab, src))
        x = torch.zeros_like(src)
        torch.cuda.synchronize()
        comm = S.TorchComm(dist)
        comm.register(work, x)
        calls = [0]
        orig = comm.exchange_tensors
        comm.exchange_tensors = lambda *a: (calls.__setitem__(0, calls[0] + 1), orig(*a))
        links = S.PeerLinks(dist, work, x, x)
        B.ok_slab_set_peers(links.struct)
        st, it, res = B.ok_slab_bicgstab([W], [src], [x], tol, 2000, comm=comm.struct, raise_on_fail=False)
        B.ok_slab_set_peers(None)
        assert comm.error is None and links.error is None, (comm.error, links.error)
        canon = torch.empty((Tl * dims[0] * dims[1] * dims[2], 12), dtype=cdtype(prec), device=DEV)
        B.ok_unpack_spinor(plocal, S.interior(slab, x), canon)
        torch.cuda.synchronize()
        results.put((rank, (st, it, res, calls[0], canon.cpu().numpy()), None))
        dist.barrier()
        del links
        dist.barrier()
        dist.destroy_process_group()
    except Exception:  # pragma: no cover
        import traceback
        results.put((rank, None, traceback.format_exc()))
