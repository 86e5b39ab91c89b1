"""Host-side logic of the t-slab decomposition that needs no GPU:
the cutting of canonical arrays into slabs and the two ok_comm callbacks over torch.distributed, run with world_size 2 on
gloo.  The per-slab apply is stood in for by the ORACLE restricted to the slab's sites, so the test fails if a halo slice
goes to the wrong neighbour, the wrong end, or is not cyclic; the reduction test checks the fixed global slab order."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle.ok_oracle import Oracle  # noqa: E402
from paper_1311_5029_b200 import inputs as I  # noqa: E402
from paper_1311_5029_b200 import slab as S  # noqa: E402

DIMS = (4, 4, 2, 8)          # 32 sites per time slice


def test_slab_ranges_and_windows():
    assert S.slab_ranges(8, 4) == [(0, 2), (2, 2), (4, 2), (6, 2)]
    U = I.near_identity_links(DIMS, 0.3, 1)
    sl = DIMS[0] * DIMS[1] * DIMS[2]
    w = S.link_window(U, DIMS, 6, 2)                      # global slices 4, 5, 6, 7, 0, 1
    assert w.shape == (6 * sl, 4, 3, 3)
    Ut = U.reshape(8, sl, 4, 3, 3)
    for k, t in enumerate([4, 5, 6, 7, 0, 1]):
        assert np.array_equal(w.reshape(6, sl, 4, 3, 3)[k], Ut[t])
    psi = I.gaussian_spinor(DIMS, 2)
    assert np.array_equal(S.spinor_slab(psi, DIMS, 2, 2), psi.reshape(8, sl, 12)[2:4].reshape(-1, 12))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, nslab, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    comm = S.TorchComm(dist)
    T, sl = DIMS[3], DIMS[0] * DIMS[1] * DIMS[2]
    U = I.near_identity_links(DIMS, 0.3, 1)
    o = Oracle(U, I.make_params(DIMS, 0.10, 0.95))
    psi = I.gaussian_spinor(DIMS, 2)
    ranges = S.slab_ranges(T, nslab * world)[rank * nslab:(rank + 1) * nslab]      # consecutive slabs on consecutive ranks
    # extended canonical fields [halo | Tloc slices | halo] of this rank's slabs, in ONE registered buffer (as the solver's workspace)
    Tl = ranges[0][1]
    buf = torch.zeros(nslab * (Tl + 2) * sl * 12, dtype=torch.complex128)
    ext = buf.view(nslab, Tl + 2, sl * 12)
    for i, (t0, _) in enumerate(ranges):
        ext[i, 1:Tl + 1] = torch.from_numpy(S.spinor_slab(psi, DIMS, t0, Tl).reshape(Tl, sl * 12))
    for i in range(nslab - 1):      # between the slabs of one process: plain copies (what ok_slab_bicgstab does on the device)
        ext[i, Tl + 1] = ext[i + 1, 1]
        ext[i + 1, 0] = ext[i, Tl]
    # the outer faces go through the C callback signature: raw addresses inside a registered buffer
    raw = buf.view(torch.uint8)
    comm.register(raw)
    nb = sl * 12 * 16
    addr = lambda i, k: raw.data_ptr() + ((i * (Tl + 2) + k) * nb)
    rc = comm._exchange(None, addr(0, 1), addr(nslab - 1, Tl), addr(0, 0), addr(nslab - 1, Tl + 1), nb)
    assert rc == 0, comm.error
    # every slab's apply from its own slices + halos only == the oracle's apply of the whole field on those sites
    err = 0.0
    parts = []
    for i, (t0, _) in enumerate(ranges):
        local = np.zeros((T, sl, 12), dtype=np.complex128)
        e = ext[i].numpy().reshape(Tl + 2, sl, 12)
        for k in range(Tl + 2):
            local[(t0 - 1 + k) % T] = e[k]
        idx = np.arange(t0 * sl, (t0 + Tl) * sl)
        got = o.apply_W(local.reshape(-1, 12), idx=idx)
        want = o.apply_W(psi, idx=idx)
        err = max(err, float(np.abs(got - want).max()))
        parts.append([float(np.vdot(psi[idx], want).real), float(np.vdot(psi[idx], want).imag), float(np.linalg.norm(want) ** 2)])
    # reduction: per-slab totals -> all-gather (C callback signature) -> sum in global slab order
    red = torch.zeros(3 * nslab * (1 + world), dtype=torch.float64)
    red[:3 * nslab] = torch.tensor(parts, dtype=torch.float64).reshape(-1)
    rraw = red.view(torch.uint8)
    comm.register(rraw)
    rc = comm._allgather(None, rraw.data_ptr(), rraw.data_ptr() + 8 * 3 * nslab, 3 * nslab)
    assert rc == 0, comm.error
    allp = red[3 * nslab:].reshape(world * nslab, 3).numpy()
    tot = [0.0, 0.0, 0.0]
    for row in allp:                       # fixed order, as k_slab_scalars
        for c in range(3):
            tot[c] += row[c]
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, err, tot, allp.tolist()))


def _run(nslab):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, nslab, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = {r: rest for r, *rest in (q.get(timeout=180) for _ in ps)}
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    return res


def test_halo_exchange_and_ordered_reduction_gloo_world2():
    U = I.near_identity_links(DIMS, 0.3, 1)
    o = Oracle(U, I.make_params(DIMS, 0.10, 0.95))
    psi = I.gaussian_spinor(DIMS, 2)
    sl = DIMS[0] * DIMS[1] * DIMS[2]
    out = o.apply_W(psi)
    for nslab in (1, 2):                   # 2 and 4 slabs in all
        res = _run(nslab)
        assert res[0][0] < 1e-13 and res[1][0] < 1e-13          # halos came from the right neighbours (cyclic in t)
        assert res[0][1] == res[1][1]                            # identical totals on both ranks, bit for bit
        assert res[0][2] == res[1][2]
        Tl = DIMS[3] // (2 * nslab)
        want = []
        for s in range(2 * nslab):         # global slab order
            idx = np.arange(s * Tl * sl, (s + 1) * Tl * sl)
            want.append([float(np.vdot(psi[idx], out[idx]).real), float(np.vdot(psi[idx], out[idx]).imag), float(np.linalg.norm(out[idx]) ** 2)])
        assert np.allclose(res[0][2], want, rtol=1e-13, atol=1e-13)
        assert abs(res[0][1][2] - np.linalg.norm(out) ** 2) <= 1e-12 * np.linalg.norm(out) ** 2
