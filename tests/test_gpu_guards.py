"""Out-of-bounds writes would not show up in a parity check (the neighbouring bytes belong to someone else), so every buffer the
hot path WRITES is placed between two guard zones here -- W in every storage format and in the 12-RHS tile layout, the
workspace, the output spinor -- on lattices whose last 32-site block is ragged, and the guards must come back untouched.
(compute-sanitizer is not available on the GPU pool; this is the bounds check the library can carry itself.)"""
import numpy as np
import pytest
import torch

import okgpu as G
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I

pytestmark = pytest.mark.gpu

GUARD = 1 << 16
PATTERN = 0xA5


def guarded(nbytes):
    """(whole buffer, the inner view of nbytes bytes); the inner view starts 256-byte aligned."""
    whole = torch.full((int(nbytes) + 2 * GUARD,), PATTERN, dtype=torch.uint8, device=G.DEV)
    assert whole.data_ptr() % 256 == 0
    return whole, whole[GUARD:GUARD + int(nbytes)]


def intact(whole, nbytes):
    torch.cuda.synchronize()
    lo, hi = whole[:GUARD], whole[GUARD + int(nbytes):]
    return bool((lo == PATTERN).all().item()) and bool((hi == PATTERN).all().item())


CASES = [(B.OK_FP32, 1, B.OK_W_DENSE), (B.OK_FP64, 1, B.OK_W_DENSE), (B.OK_FP32, 1, B.OK_W_BLOCK), (B.OK_FP32, 1, B.OK_W_DS),
         (B.OK_FP64, 1, B.OK_W_CONJ), (B.OK_FP32, 1, B.OK_W_PAULI), (B.OK_FP64, 1, B.OK_W_PAULI), (B.OK_FP32, 12, B.OK_W_DENSE)]


@pytest.mark.parametrize("dims", [(4, 3, 3, 2), (6, 5, 2, 3), (4, 4, 4, 8)])
@pytest.mark.parametrize("prec,nrhs,storage", CASES)
def test_precalc_apply_and_solver_write_only_what_they_own(dims, prec, nrhs, storage):
    U = I.near_identity_links(dims, 0.3, 1)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    p = B.make_params(pd, prec, nrhs=nrhs, storage=storage)
    wb, vb, kb = B.ok_W_bytes(p), B.ok_vec_bytes(p), B.ok_work_bytes(p)
    Wall, W = guarded(wb)
    Kall, work = guarded(kb)
    B.ok_set_stream(None)
    B.ok_set_workspace(work, kb)
    try:
        B.ok_precalc_W(G.to_dev(U, torch.complex128), p, W)
        assert intact(Wall, wb) and intact(Kall, kb)
        V = int(np.prod(dims))
        shape = (V, 12) if nrhs == 1 else (V, 12, 12)
        rng = np.random.default_rng(3)
        psi = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        Sall, src = guarded(vb)
        src.zero_()
        B.ok_pack_spinor(p, G.to_dev(psi, G.cdtype(prec)), src)
        Oall, out = guarded(vb)
        B.ok_dirac_apply(W, src, out)
        assert intact(Oall, vb) and intact(Sall, vb) and intact(Wall, wb)
        Xall, x = guarded(vb)
        st, it, res = B.ok_bicgstab(W, src, x, 1e-5 if prec == B.OK_FP32 else 1e-10, 500)
        assert st == 0 and res <= (1e-5 if prec == B.OK_FP32 else 1e-10)
        assert intact(Xall, vb) and intact(Kall, kb) and intact(Sall, vb) and intact(Wall, wb)
        if nrhs == 1:
            Rall, result = guarded(24)
            B.ok_dirac_apply_dot_static(W, src, x, out, result)
            assert intact(Rall, 24) and intact(Oall, vb)
    finally:
        torch.cuda.synchronize()
        B.lib().ok_forget_W(W.data_ptr())
        B.ok_set_workspace(None)
