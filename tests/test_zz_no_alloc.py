"""ok_dirac_apply_dot_static (ok.h): the entry point that allocates nothing -- its scratch is a static __device__ array inside
the library.  Checked against the existing path (ok_dirac_apply for out, fp64 sums over that output for the three
reductions) on two calls in a row: the second on a smaller lattice and another W format, so that the rows the first call
left in the shared array lie beyond what the second one may read.  Collected last (file name) so that a failure here hides
no other test under `pytest -x`; needs nothing from the tests before it."""
import ctypes as C

import numpy as np
import pytest
import torch

import okgpu as G
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _setup(dims, prec, storage, seed):
    U = I.near_identity_links(dims, 0.3, seed)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    p = B.make_params(pd, prec, storage=storage)
    W = G.precalc(p, U)
    psi = G.pack_spinor(p, I.gaussian_spinor(dims, seed + 1))
    a = G.pack_spinor(p, I.gaussian_spinor(dims, seed + 2))
    return p, W, psi, a


def _fields(p, t):
    """packed spinor buffer -> flat fp64 complex tensor (padding lanes are zero in both operands of every sum below)"""
    real = torch.float64 if p.precision == B.OK_FP64 else torch.float32
    r = t.view(real).to(torch.float64).reshape(-1, 2)
    return torch.complex(r[:, 0], r[:, 1])


def _check(p, W, psi, a, tol):
    want = B.alloc_vec(p, G.DEV)
    B.ok_dirac_apply(W, psi, want)                       # the existing path
    got = B.alloc_vec(p, G.DEV)
    got.fill_(0x5A)                                      # the call must write every byte it owns
    result = torch.full((3,), float("nan"), dtype=torch.float64, device=G.DEV)
    B.ok_dirac_apply_dot_static(W, psi, a, got, result)
    torch.cuda.synchronize()
    first = result.clone()
    # once the kernels are loaded, a call leaves the device's free memory as it was: nothing is allocated (or freed) by it
    free0 = torch.cuda.mem_get_info()[0]
    B.ok_dirac_apply_dot_static(W, psi, a, got, result)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.equal(first, result)                    # same bits from the shared scratch array the second time
    w, g_, av = _fields(p, want), _fields(p, got), _fields(p, a)
    # internal layout: the element order inside a block differs from the canonical one, but it is the same for a and out
    err = (torch.linalg.vector_norm(g_ - w) / torch.linalg.vector_norm(w)).item()
    assert err <= tol, err
    dot = torch.sum(torch.conj(av) * w)
    nrm2 = torch.sum(w.real ** 2 + w.imag ** 2).item()
    scale = (torch.linalg.vector_norm(av) * torch.linalg.vector_norm(w)).item()
    r = result.cpu().numpy()
    assert np.all(np.isfinite(r))
    assert abs(r[0] - dot.real.item()) <= tol * scale
    assert abs(r[1] - dot.imag.item()) <= tol * scale
    assert abs(r[2] - nrm2) <= tol * nrm2
    return r


def test_two_calls_in_a_row_match_the_existing_path():
    # first call: 8^3 x 16 fp64 dense (256 blocks of partial sums)
    p1, W1, psi1, a1 = _setup((8, 8, 8, 16), B.OK_FP64, B.OK_W_DENSE, 11)
    r1 = _check(p1, W1, psi1, a1, 1e-12)
    # second call right after it: a ragged 4 x 3 x 3 x 2 lattice (72 sites, 3 blocks), fp32, the Pauli format
    p2, W2, psi2, a2 = _setup((4, 3, 3, 2), B.OK_FP32, B.OK_W_PAULI, 21)
    r2 = _check(p2, W2, psi2, a2, 2e-5)
    assert r1[2] > 10 * r2[2]                             # stale rows of the first call would have dominated the second sum
    # and the first problem again: bit-identical result (fixed summation order, no state carried between calls)
    r3 = _check(p1, W1, psi1, a1, 1e-12)
    assert np.array_equal(r1, r3)


def test_sizes_beyond_the_static_array_are_rejected():
    assert B.ok_static_max_sites() == 2097152
    # a W header that describes a lattice of 2^22 sites (no payload behind it: the call must refuse before touching any)
    p, W, psi, a = _setup((4, 4, 4, 8), B.OK_FP32, B.OK_W_DENSE, 31)
    hdr = W[:1024].clone().cpu().numpy()
    big = B.ok_params.from_buffer_copy(hdr[8:8 + C.sizeof(B.ok_params)].tobytes())
    assert list(big.dims) == [4, 4, 4, 8]
    big.dims[:] = [64, 64, 32, 32]
    hdr[8:8 + C.sizeof(B.ok_params)] = np.frombuffer(bytes(big), dtype=np.uint8)
    fake = torch.from_numpy(hdr).to(G.DEV)
    out = B.alloc_vec(p, G.DEV)
    result = torch.zeros(3, dtype=torch.float64, device=G.DEV)
    try:
        with pytest.raises(B.OkError) as e:
            B.ok_dirac_apply_dot_static(fake, psi, a, out, result)
        assert e.value.status == -1
        assert "OK_STATIC_MAX_SITES" in str(e.value) and "4194304" in str(e.value)
    finally:
        B.lib().ok_forget_W(fake.data_ptr())
    torch.cuda.synchronize()
    # the library is still usable afterwards
    _check(p, W, psi, a, 2e-5)
