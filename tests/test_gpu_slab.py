"""t-slab decomposition on the device (include/ok.h ok_slab_*): several slabs
held by one process stand in for the ranks ("virtual ranks": separate W, fields and halos per slab).
  * ok_slab_precalc_W from a slab's link window == the whole-lattice W on the slab's sites, bit for bit;
  * ok_slab_dirac_apply with the neighbours' boundary slices in the halos == the whole-lattice apply, bit for bit, and
    within the north_star tolerance of the ORACLE on the full lattice;
  * ok_slab_dirac_apply_peer (halo exchange fused into the apply: the neighbours' boundary slices loaded in place) the same, with
    the neighbours in this process and in ANOTHER process whose memory is mapped through CUDA IPC;
  * ok_slab_bicgstab == the oracle's BiCGStab (iterations +-2, true residual <= tol, solution), bit-reproducible, and
    bit-identical whether the T closure is read in place or goes through the ok_comm callbacks (the multi-process path).
"""
import numpy as np
import pytest
import torch

from oracle import ok_oracle as oo
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
from paper_1311_5029_b200 import slab as S
import okgpu as G

pytestmark = pytest.mark.gpu

CASES = [((4, 4, 4, 8), 2), ((4, 4, 4, 8), 4), ((4, 4, 2, 16), 4), ((8, 4, 2, 12), 2)]


def setup(dims, eps=0.3, seed=1, bc=None):
    U = I.near_identity_links(dims, eps, seed)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    if bc is not None:
        pd["bc"] = bc
    return U, pd, oo.Oracle(U, pd)


class Slabs:
    """nslab slabs of one lattice on the device: W per slab, workspace, helpers to scatter / gather canonical fields."""

    def __init__(self, U, pd, prec, nslab):
        self.dims, self.prec, self.nslab = tuple(pd["dims"]), prec, nslab
        self.p = B.make_params(pd, prec)
        self.ranges = S.slab_ranges(self.dims[3], nslab)
        self.slab = B.make_slab_params(self.p, self.ranges[0][1])
        self.work = B.alloc_bytes(B.ok_slab_work_bytes(self.slab, nslab, 1), G.DEV)
        B.ok_set_stream(None)
        B.ok_set_workspace(self.work, self.work.numel())
        self.W = []
        for t0, Tl in self.ranges:
            W = B.alloc_W(self.slab, G.DEV)
            B.ok_slab_precalc_W(G.to_dev(S.link_window(U, self.dims, t0, Tl), torch.complex128), self.slab, self.dims[3], t0, W)
            self.W.append(W)
        torch.cuda.synchronize()
        self.plocal = B.make_params(dict(pd, dims=self.dims[:3] + (self.ranges[0][1],)), prec)

    def scatter(self, psi):
        """canonical [V][12] -> one extended device field per slab (halos zero)."""
        out = []
        for t0, Tl in self.ranges:
            v = torch.zeros(B.ok_slab_vec_bytes(self.slab), dtype=torch.uint8, device=G.DEV)
            B.ok_pack_spinor(self.plocal, G.to_dev(S.spinor_slab(psi, self.dims, t0, Tl), G.cdtype(self.prec)), S.interior(self.slab, v))
            out.append(v)
        return out

    def fill_halos(self, vecs):
        n = self.nslab
        for i in range(n):
            lo, first, last, hi = S.halo_views(self.slab, vecs[i])
            lo.copy_(S.halo_views(self.slab, vecs[(i - 1) % n])[2])
            hi.copy_(S.halo_views(self.slab, vecs[(i + 1) % n])[1])

    def gather(self, vecs):
        parts = []
        for v in vecs:
            Tl = self.slab.dims[3]
            canon = torch.empty((Tl * self.dims[0] * self.dims[1] * self.dims[2], 12), dtype=G.cdtype(self.prec), device=G.DEV)
            B.ok_unpack_spinor(self.plocal, S.interior(self.slab, v), canon)
            parts.append(canon)
        torch.cuda.synchronize()
        return torch.cat(parts).cpu().numpy().astype(np.complex128)


@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims,nslab", CASES)
def test_slab_W_and_apply_equal_the_whole_lattice_bit_for_bit(dims, nslab, prec):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    Wc = G.unpack_W(p, W, o.V)
    sl = Slabs(U, pd, prec, nslab)
    sites = dims[0] * dims[1] * dims[2]
    for (t0, Tl), Ws in zip(sl.ranges, sl.W):
        got = G.unpack_W(sl.plocal, Ws, Tl * sites)
        assert np.array_equal(got, Wc[t0 * sites:(t0 + Tl) * sites])               # incl. the antiperiodic sign where T - 1 falls
    psi = I.gaussian_spinor(dims, 2)
    whole = G.apply(p, W, psi)
    vecs = sl.scatter(psi)
    sl.fill_halos(vecs)
    outs = [torch.zeros_like(v) for v in vecs]
    for Ws, v, out in zip(sl.W, vecs, outs):
        B.ok_slab_dirac_apply(Ws, v, out)
    got = sl.gather(outs)
    assert np.array_equal(got, whole)
    want = o.apply_W(psi)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= 1e-12
    else:
        assert G.rel_l2(got, want) <= 2e-5
    B.ok_set_workspace(None)


@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims,nslab", CASES)
def test_slab_apply_with_fused_halo_loads_equals_the_whole_lattice_bit_for_bit(dims, nslab, prec):
    """ok_slab_dirac_apply_peer: the neighbours' boundary slices are read in place (the address a peer GPU's mapped buffer would
    have); this slab's own halo slices are poisoned to show that nothing reads them."""
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    psi = I.gaussian_spinor(dims, 2)
    whole = G.apply(p, W, psi)
    sl = Slabs(U, pd, prec, nslab)
    vecs = sl.scatter(psi)
    for v in vecs:
        lo, first, last, hi = S.halo_views(sl.slab, v)
        lo.fill_(0xFF)          # NaN patterns in both precisions
        hi.fill_(0xFF)
    outs = [torch.zeros_like(v) for v in vecs]
    for i, (Ws, v, out) in enumerate(zip(sl.W, vecs, outs)):
        lo_slice = S.halo_views(sl.slab, vecs[(i - 1) % nslab])[2]      # the lower neighbour's last own slice
        hi_slice = S.halo_views(sl.slab, vecs[(i + 1) % nslab])[1]      # the upper neighbour's first own slice
        B.ok_slab_dirac_apply_peer(Ws, v, lo_slice, hi_slice, out)
    got = sl.gather(outs)
    assert np.array_equal(got, whole)
    want = o.apply_W(psi)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= 1e-12
    else:
        assert G.rel_l2(got, want) <= 2e-5
    with pytest.raises(B.OkError):
        B.ok_slab_dirac_apply_peer(sl.W[0], vecs[0], None, S.halo_views(sl.slab, vecs[0])[1], outs[0])
    B.ok_set_workspace(None)


def test_slab_apply_reads_another_process_memory_through_cuda_ipc():
    """Two processes on cuda:0, one slab each: every process maps the other's field through CUDA IPC and its apply loads the
    neighbour's boundary slices straight from that mapping -- the mechanism a multi-GPU run uses over NVLink peer access --
    and the gathered result equals the whole-lattice apply bit for bit."""
    import torch.multiprocessing as mp
    try:   # two processes must be allowed on the one GPU (compute mode DEFAULT); anything else is an environment limit, not a failure
        import pynvml
        pynvml.nvmlInit()
        mode = pynvml.nvmlDeviceGetComputeMode(pynvml.nvmlDeviceGetHandleByIndex(torch.cuda.current_device()))
        if mode != pynvml.NVML_COMPUTEMODE_DEFAULT:
            pytest.skip("GPU compute mode %d does not admit a second process" % mode)
    except Exception:   # no NVML: go on (pytest.skip is a BaseException and passes through)
        pass
    dims, nranks, prec = (4, 4, 4, 8), 2, B.OK_FP64
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec)
    psi = I.gaussian_spinor(dims, 2)
    whole = G.apply(p, G.precalc(p, U), psi)
    ctx = mp.get_context("spawn")
    q_in = [ctx.Queue() for _ in range(nranks)]
    results, barrier = ctx.Queue(), ctx.Barrier(nranks)
    procs = [ctx.Process(target=G.ipc_slab_worker, args=(r, nranks, U, pd, prec, psi, q_in, q_in, results, barrier)) for r in range(nranks)]
    for pr in procs:
        pr.start()
    try:
        parts = {}
        for _ in range(nranks):
            rank, arr, err = results.get(timeout=300)
            assert err is None, err
            parts[rank] = arr
    finally:
        for pr in procs:
            pr.join(timeout=60)
            if pr.is_alive():
                pr.kill()
    got = np.concatenate([parts[r] for r in range(nranks)]).astype(np.complex128)
    assert np.array_equal(got, whole)
    B.ok_set_workspace(None)


def test_slab_bicgstab_with_peer_access_across_two_processes():
    """ok_slab_set_peers: two processes on cuda:0, one slab each; in every apply of the solver each process reads the other's
    boundary slices (of p, s and x) in place through CUDA IPC mappings of the other's workspace and x buffer; `exchange` is never
    called.  Bit-identical to the two-slab solve of one process."""
    import torch.multiprocessing as mp
    try:
        import pynvml
        pynvml.nvmlInit()
        mode = pynvml.nvmlDeviceGetComputeMode(pynvml.nvmlDeviceGetHandleByIndex(torch.cuda.current_device()))
        if mode != pynvml.NVML_COMPUTEMODE_DEFAULT:
            pytest.skip("GPU compute mode %d does not admit a second process" % mode)
    except Exception:
        pass
    dims, nranks, prec, tol = (4, 4, 4, 8), 2, B.OK_FP64, 1e-10
    U, pd, o = setup(dims)
    b = I.gaussian_spinor(dims, 2)
    sl = Slabs(U, pd, prec, nranks)
    src = sl.scatter(b)
    xs = [torch.zeros_like(v) for v in src]
    want = B.ok_slab_bicgstab(sl.W, src, xs, tol, 2000, raise_on_fail=False)
    xwant = sl.gather(xs)
    B.ok_set_workspace(None)
    ctx = mp.get_context("spawn")
    q_in, q_ag = [ctx.Queue() for _ in range(nranks)], [ctx.Queue() for _ in range(nranks)]
    results, barrier = ctx.Queue(), ctx.Barrier(nranks)
    procs = [ctx.Process(target=G.ipc_solver_worker, args=(r, nranks, U, pd, prec, b, tol, q_in, q_ag, results, barrier)) for r in range(nranks)]
    for pr in procs:
        pr.start()
    try:
        parts = {}
        for _ in range(nranks):
            rank, val, err = results.get(timeout=300)
            assert err is None, err
            parts[rank] = val
    finally:
        for pr in procs:
            pr.join(timeout=60)
            if pr.is_alive():
                pr.kill()
    for r in range(nranks):
        st, it, res, calls, _ = parts[r]
        assert (st, it, res) == want                                   # same iteration, same residual, on every process
        assert calls["exchange"] == 0 and calls["barrier"] >= 2 * it and calls["allgather"] >= 3 * it
    got = np.concatenate([parts[r][4] for r in range(nranks)]).astype(np.complex128)
    assert np.array_equal(got, xwant)
    # the same through the package's own plumbing: torch.distributed + slab.TorchComm + slab.PeerLinks
    import socket
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    results = ctx.Queue()
    procs = [ctx.Process(target=G.torch_peer_solver_worker, args=(r, nranks, port, U, pd, prec, b, tol, results)) for r in range(nranks)]
    for pr in procs:
        pr.start()
    try:
        parts = {}
        for _ in range(nranks):
            rank, val, err = results.get(timeout=300)
            assert err is None, err
            parts[rank] = val
    finally:
        for pr in procs:
            pr.join(timeout=60)
            if pr.is_alive():
                pr.kill()
    for r in range(nranks):
        assert parts[r][:3] == want and parts[r][3] == 0               # exchange_tensors never ran
    got = np.concatenate([parts[r][4] for r in range(nranks)]).astype(np.complex128)
    assert np.array_equal(got, xwant)


def test_slab_apply_periodic_time_and_error_paths():
    dims = (4, 4, 2, 8)
    U, pd, o = setup(dims, bc=[1, 1, 1, 1])
    sl = Slabs(U, pd, B.OK_FP64, 2)
    psi = I.gaussian_spinor(dims, 5)
    vecs = sl.scatter(psi)
    sl.fill_halos(vecs)
    outs = [torch.zeros_like(v) for v in vecs]
    for Ws, v, out in zip(sl.W, vecs, outs):
        B.ok_slab_dirac_apply(Ws, v, out)
    assert G.per_site_rel_err(sl.gather(outs), o.apply_W(psi)) <= 1e-12
    # a slab W is open in t: the whole-lattice calls refuse it, and the slab calls refuse a whole-lattice W
    with pytest.raises(B.OkError):
        B.ok_dirac_apply(sl.W[0], vecs[0], outs[0])
    p = B.make_params(pd, B.OK_FP64)
    Wfull = G.precalc(p, U)
    with pytest.raises(B.OkError):
        B.ok_slab_dirac_apply(Wfull, vecs[0], outs[0])
    bad = B.make_slab_params(B.make_params(dict(pd, dims=(3, 3, 3, 8)), B.OK_FP64), 4)       # 27 sites per slice
    assert B.ok_slab_vec_bytes(bad) == 0
    # the link window must fit the lattice once (Tloc + 4 <= T), t0 must be a slice of it, the workspace must be there
    Wt = B.alloc_W(sl.slab, G.DEV)
    lk = G.to_dev(S.link_window(U, dims, 0, 4), torch.complex128)
    for T_global, t0 in ((7, 0), (8, -1), (8, 8)):
        with pytest.raises(B.OkError) as e:
            B.ok_slab_precalc_W(lk, sl.slab, T_global, t0, Wt)
        assert e.value.status == -1
    B.ok_set_workspace(None, 0)
    with pytest.raises(B.OkError) as e:
        B.ok_slab_precalc_W(lk, sl.slab, 8, 0, Wt)
    assert e.value.status == -5
    # slabs of different precision cannot be solved together
    p32 = B.make_params(pd, B.OK_FP32)
    sl32 = Slabs(U, pd, B.OK_FP32, 2)
    v64, v32 = sl.scatter(psi), sl32.scatter(psi)
    st, _, _ = B.ok_slab_bicgstab([sl.W[0], sl32.W[1]], [v64[0], v32[1]], [torch.zeros_like(v64[0]), torch.zeros_like(v32[1])], 1e-8, 10,
                                  raise_on_fail=False)
    assert st == -1
    B.ok_set_workspace(None)


class LoopComm(S.TorchComm):
    """ok_comm of a single process (rank 0 of 1) without torch.distributed: the callbacks close the T direction on the
    process itself -- the same C code path a multi-process run takes."""

    def __init__(self):
        self.torch, self.dist, self.group, self.stream = torch, None, None, None
        self.rank, self.nranks, self.buffers, self.error = 0, 1, [], None
        self.calls = [0, 0]
        self._ex = B.EXCHANGE_FN(self._exchange)
        self._ag = B.ALLGATHER_FN(self._allgather)
        self.struct = B.ok_comm(0, 1, self._ex, self._ag, None)

    def exchange_tensors(self, *a):
        self.calls[0] += 1
        super().exchange_tensors(*a)

    def allgather_tensors(self, *a):
        self.calls[1] += 1
        super().allgather_tensors(*a)


@pytest.mark.parametrize("prec,tol", [(B.OK_FP64, 1e-10), (B.OK_FP32, 1e-6)])
@pytest.mark.parametrize("dims,nslab", CASES)
def test_slab_bicgstab_vs_oracle(dims, nslab, prec, tol):
    U, pd, o = setup(dims)
    sl = Slabs(U, pd, prec, nslab)
    b = I.gaussian_spinor(dims, 2)
    src = sl.scatter(b)
    xs = [torch.zeros_like(v) for v in src]
    st, it, res = B.ok_slab_bicgstab(sl.W, src, xs, tol, 2000, raise_on_fail=False)
    Wc = o.precalc_W()
    xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), b, tol, 2000)
    assert st == 0 and sto == 0 and abs(it - ito) <= 2 and res <= tol
    x = sl.gather(xs)
    r = b - o.apply_W(x, W=Wc)
    slack = 0.0 if prec == B.OK_FP64 else G.fp32_operator_slack(o, x, b, W=Wc)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= tol * 1.0001 + slack
    assert G.rel_l2(x, xo) <= 50 * tol
    # bit-reproducible
    xs2 = [torch.zeros_like(v) for v in src]
    assert B.ok_slab_bicgstab(sl.W, src, xs2, tol, 2000, raise_on_fail=False) == (st, it, res)
    assert all(torch.equal(S.interior(sl.slab, a), S.interior(sl.slab, c)) for a, c in zip(xs, xs2))
    # the same solve with the T closure and the reductions going through the ok_comm callbacks
    comm = LoopComm()
    comm.register(sl.work, *xs2)
    xs3 = [torch.zeros_like(v) for v in src]
    comm.register(*xs3)
    st3 = B.ok_slab_bicgstab(sl.W, src, xs3, tol, 2000, comm=comm.struct, raise_on_fail=False)
    assert comm.error is None and st3 == (st, it, res)
    assert all(torch.equal(S.interior(sl.slab, a), S.interior(sl.slab, c)) for a, c in zip(xs, xs3))
    assert comm.calls[0] >= 2 * it and comm.calls[1] >= 3 * it        # 2 halo refreshes and 3 reductions per iteration
    # the unsharded solver on the same system: same iteration count within the +-2 of the contract
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    G.workspace(p)
    xw = B.alloc_vec(p)
    stw, itw, resw = B.ok_bicgstab(W, G.pack_spinor(p, b), xw, tol, 2000, raise_on_fail=False)
    assert stw == 0 and abs(itw - it) <= 2
    assert G.rel_l2(G.unpack_spinor(p, xw, b.shape), x) <= 50 * tol
    B.ok_set_workspace(None)


def test_slab_bicgstab_edge_cases():
    dims = (4, 4, 2, 8)
    U, pd, o = setup(dims)
    sl = Slabs(U, pd, B.OK_FP64, 2)
    zero = sl.scatter(np.zeros((o.V, 12), dtype=np.complex128))
    xs = [torch.ones_like(v) for v in zero]
    st, it, res = B.ok_slab_bicgstab(sl.W, zero, xs, 1e-10, 100, raise_on_fail=False)
    assert (st, it, res) == (0, 0, 0.0) and np.all(sl.gather(xs) == 0)
    src = sl.scatter(I.gaussian_spinor(dims, 2))
    st, it, res = B.ok_slab_bicgstab(sl.W, src, xs, 1e-10, 3, raise_on_fail=False)
    assert st == -4 and it == 3 and res > 1e-10
    B.ok_set_workspace(None, 0)
    with pytest.raises(B.OkError) as e:
        B.ok_slab_bicgstab(sl.W, src, xs, 1e-10, 100)
    assert e.value.status == -5
