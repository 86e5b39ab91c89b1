"""OK_W_PAULI ("compress the 432 color blocks into 50"): the Pauli components of the
D and S blocks of W^0 and the 13 positive-direction matrices, 49 colour blocks by the structure of Eqs. (2.6)-(2.12), 37
stored matrices per site once components that coincide up to a constant of the action are merged (csrc/ok_pauli.cu).
Same operator as the dense Eq. (2.2) form, so the oracle side is unchanged: Oracle.precalc_W / apply_W / bicgstab; the
tolerances are the dense path's (fp64 per-site 1e-12, fp32 relative L2 2e-5, iterations +-2)."""
import numpy as np
import pytest
import torch

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu

SHAPES = [(4, 3, 3, 2), (2, 2, 2, 2), (4, 4, 4, 8), (5, 2, 3, 4), (8, 4, 2, 6)]


def setup(dims, eps=0.3, seed=1, kappa=0.10, bc=(1, 1, 1, -1), haar=False, coeffs=None):
    U = I.haar_links(dims, seed) if haar else I.near_identity_links(dims, eps, seed)
    u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
    pd = I.make_params(dims, kappa, u0, bc=bc, coeffs=coeffs)
    return U, pd, Oracle(U, pd)


@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_pauli_precalc_W_and_apply(dims, prec):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec, storage=B.OK_W_PAULI)
    V = o.V
    assert B.ok_W_bytes(p) == 1024 + ((V + 31) // 32) * 32 * 37 * 9 * (16 if prec == B.OK_FP64 else 8)
    W = G.precalc(p, U)
    q = B.ok_W_params(W)
    assert list(q.dims) == list(dims) and q.storage == B.OK_W_PAULI and q.precision == prec
    # the 27 dense matrices rebuilt from the 37 stored ones (ok_unpack_W) against the oracle's W, element by element.
    # fp32: an entry is a sum of up to two stored (once-rounded) components: 2 x 2^-24 relative to the largest
    want_W = o.precalc_W()
    got_W = G.unpack_W(p, W, V)
    tolW = 2e-13 if prec == B.OK_FP64 else 4e-7
    assert np.abs(got_W - want_W).max() <= tolW * np.abs(want_W).max()
    assert np.all(got_W[want_W == 0] == 0)                 # the 172 structurally zero colour blocks stay exactly zero
    psi = I.gaussian_spinor(dims, 2)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi, W=want_W)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= 1e-12
    else:
        assert G.rel_l2(got, want) <= 2e-5
    assert np.all(G.apply(p, W, np.zeros_like(psi)) == 0)
    # padded lanes of the last 32-site block stay zero in the internal layout
    packed_out = B.alloc_vec(p)
    B.ok_dirac_apply(W, G.pack_spinor(p, psi), packed_out)
    torch.cuda.synchronize()
    raw = packed_out.view(torch.float64 if prec == B.OK_FP64 else torch.float32).cpu().numpy()
    nblk = (V + 31) // 32
    units = raw.reshape(nblk, -1, 32, 2 if prec == B.OK_FP64 else 4)
    if V % 32:
        assert np.all(units[-1, :, V % 32:, :] == 0)
    # only ok_precalc_W writes this format
    with pytest.raises(B.OkError):
        B.ok_pack_W(p, G.to_dev(want_W, G.cdtype(prec)), W)


@pytest.mark.parametrize("case", ["haar", "periodic", "mixed-bc", "wilson", "u0=1"])
def test_pauli_variants(case):
    dims = (4, 4, 4, 8) if case == "haar" else (4, 3, 3, 4)
    U, pd, o = setup(dims, haar=case == "haar", kappa=0.08 if case == "haar" else 0.10,
                     bc={"periodic": (1, 1, 1, 1), "mixed-bc": (-1, 1, -1, -1)}.get(case, (1, 1, 1, -1)),
                     coeffs=I.WILSON if case == "wilson" else None)
    if case == "u0=1":
        pd["u0"] = 1.0
        o = Oracle(U, pd)
    p = B.make_params(pd, B.OK_FP64, storage=B.OK_W_PAULI)
    W = G.precalc(p, U)
    want_W = o.precalc_W()
    assert np.abs(G.unpack_W(p, W, o.V) - want_W).max() <= 2e-13 * np.abs(want_W).max()
    psi = I.gaussian_spinor(dims, 4)
    assert G.per_site_rel_err(G.apply(p, W, psi), o.apply_W(psi, W=want_W)) <= 1e-12
    # identical to the dense CUDA path to rounding order
    pdn = B.make_params(pd, B.OK_FP64)
    assert G.rel_l2(G.apply(p, W, psi), G.apply(pdn, G.precalc(pdn, U), psi)) <= 1e-14


@pytest.mark.parametrize("prec,tol", [(B.OK_FP64, 1e-10), (B.OK_FP32, 1e-6)])
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 3, 3, 2)])
def test_pauli_bicgstab_and_cgnr_vs_oracle(dims, prec, tol):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec, storage=B.OK_W_PAULI)
    W = G.precalc(p, U)
    b = I.gaussian_spinor(dims, 2)
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    st, it, res = B.ok_bicgstab(W, src, x, tol, 2000, raise_on_fail=False)
    assert st == 0 and res <= tol
    Wc = o.precalc_W()
    xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), b, tol, 2000)
    assert sto == 0 and abs(it - ito) <= 2
    xs = G.unpack_spinor(p, x, b.shape)
    r = b - o.apply_W(xs, W=Wc)
    # R-RESID; this format rounds the Pauli components, an entry of W is a sum of up to two of them: 2 units more
    slack = 0.0 if prec == B.OK_FP64 else 2 * G.fp32_operator_slack(o, xs, b, W=Wc)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= tol * 1.0001 + slack
    x2 = B.alloc_vec(p)
    assert B.ok_bicgstab(W, src, x2, tol, 2000, raise_on_fail=False) == (st, it, res) and torch.equal(x, x2)     # bit-reproducible
    stc, itc, resc = B.ok_cgnr(W, src, x2, tol, 5000, raise_on_fail=False)
    assert stc == 0 and resc <= tol
