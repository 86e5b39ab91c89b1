"""ok_dirac_apply_host (include/ok.h): Eq. (2.2), with HOST spinors in the canonical layout -- the e2e leg of
bench.py.  Lattices with T >= 8 and a 32-aligned time slice take the pipelined path (chunks of time slices applied behind the
host -> device copy, 4 / 8 / 16 chunks); the others the sequential one.  Both must equal ok_dirac_apply bit for bit and match
the oracle within the north_star tolerances."""
import numpy as np
import pytest
import torch

from oracle import ok_oracle as oo
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 4, 2, 16), (4, 4, 2, 36), (4, 4, 2, 9), (4, 3, 3, 2), (3, 3, 3, 8)])
@pytest.mark.parametrize("pinned", [True, False])
@pytest.mark.parametrize("pipeline", [True, False])
def test_host_apply_equals_device_apply_and_oracle(dims, prec, pinned, pipeline, monkeypatch):
    # fields below 8 MiB take the sequential path unless OK_HOST_PIPELINE is set (include/ok.h); both are exercised here
    if pipeline:
        monkeypatch.setenv("OK_HOST_PIPELINE", "1")
    else:
        monkeypatch.delenv("OK_HOST_PIPELINE", raising=False)
    U = I.near_identity_links(dims, 0.3, 1)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    o = oo.Oracle(U, pd)
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    psi = I.gaussian_spinor(dims, 2)
    want_dev = G.apply(p, W, psi)
    G.workspace(p)
    hin = torch.from_numpy(psi).to(G.cdtype(prec))
    hout = torch.full_like(hin, float("nan"))
    if pinned:
        hin, hout = hin.pin_memory(), hout.pin_memory()
    for _ in range(2):          # twice: the library-owned copy streams and events are reused
        B.ok_dirac_apply_host(W, hin, hout)
    got = hout.numpy().astype(np.complex128)
    assert np.array_equal(got, want_dev)
    want = o.apply_W(psi)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= 1e-12
    else:
        assert G.rel_l2(got, want) <= 2e-5


def test_host_apply_12rhs():
    dims = (4, 4, 4, 8)
    U = I.near_identity_links(dims, 0.3, 1)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    o = oo.Oracle(U, pd)
    p = B.make_params(pd, B.OK_FP32, nrhs=12)
    W = G.precalc(p, U)
    psi = np.stack([I.gaussian_spinor(dims, 30 + j) for j in range(12)], axis=2)
    G.workspace(p)
    hin = torch.from_numpy(psi).to(torch.complex64).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    B.ok_dirac_apply_host(W, hin, hout)
    got = hout.numpy().astype(np.complex128)
    want = o.apply_W(psi)
    num = np.linalg.norm((got - want).reshape(-1, 12), axis=0)
    den = np.linalg.norm(want.reshape(-1, 12), axis=0)
    assert float((num / den).max()) <= 2e-5
