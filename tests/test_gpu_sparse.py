"""Parity of the reduced W storage formats with the CPU oracle.

OK_W_BLOCK keeps the 260 structurally non-zero colour blocks of a site (432 blocks, 172 vanish),
OK_W_DS keeps D and S of W = [[D, S], [+-S, D]] once per term (Eqs. 2.6-2.12), OK_W_CONJ keeps them for
W^0 and the positive-direction terms only and rebuilds the opposite directions from the neighbour site by the conjugation
relations (Eqs. 2.3, 2.10; the paper's own compression).  All hold the same
operator as the dense Eq. (2.2) form, so the oracle side is unchanged: Oracle.precalc_W / apply_W / bicgstab.
Tolerances as for the dense path (fp64 per-site 1e-12, fp32 relative L2 2e-5, iterations +-2).
"""
import numpy as np
import pytest
import torch

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu

FP64_TOL = 1e-12
FP32_TOL = 2e-5
SHAPES = [(4, 3, 3, 2), (2, 2, 2, 2), (4, 4, 4, 8), (5, 2, 3, 4)]
FORMATS = [B.OK_W_BLOCK, B.OK_W_DS, B.OK_W_CONJ]
BLOCKS = {B.OK_W_BLOCK: 260, B.OK_W_DS: 132, B.OK_W_CONJ: 70}


def setup(dims, eps=0.3, seed=1, kappa=0.10, bc=(1, 1, 1, -1), haar=False):
    U = I.haar_links(dims, seed) if haar else I.near_identity_links(dims, eps, seed)
    u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
    pd = I.make_params(dims, kappa, u0, bc=bc)
    return U, pd, Oracle(U, pd)


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_sparse_pack_unpack_and_apply_with_oracle_W(dims, prec, fmt):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec, storage=fmt)
    V = o.V
    assert B.ok_W_bytes(p) == 1024 + ((V + 31) // 32) * 32 * BLOCKS[fmt] * 9 * (16 if prec == B.OK_FP64 else 8)
    Wc = o.precalc_W()
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wc, G.cdtype(prec)), W)
    back = G.unpack_W(p, W, V)
    # the oracle's W has exactly the structure both formats rely on: the round trip loses nothing but the rounding to `prec`
    assert np.array_equal(back.astype(G.npdtype(prec)), Wc.astype(G.npdtype(prec)))
    q = B.ok_W_params(W)
    assert list(q.dims) == list(dims) and q.storage == fmt and q.precision == prec
    psi = I.gaussian_spinor(dims, 2)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi, W=Wc)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= FP64_TOL
    else:
        assert G.rel_l2(got, want) <= FP32_TOL
    # same answer as the dense CUDA path on the same W (fp64: to rounding order)
    pdn = B.make_params(pd, prec)
    Wd = B.alloc_W(pdn)
    B.ok_pack_W(pdn, G.to_dev(Wc, G.cdtype(prec)), Wd)
    dense = G.apply(pdn, Wd, psi)
    assert G.rel_l2(got, dense) <= (1e-14 if prec == B.OK_FP64 else 2e-6)


@pytest.mark.parametrize("fmt", FORMATS)
def test_block_format_keeps_any_matrix_with_the_zero_pattern(fmt):
    """OK_W_BLOCK stores every quadrant on its own: a random W with the structural zero pattern survives the round trip;
    OK_W_DS keeps UL (else LR) and UR and rebuilds the rest from them."""
    dims = (4, 3, 3, 2)
    U, pd, o = setup(dims)
    V = o.V
    pattern = np.abs(o.precalc_W()).max(axis=0) > 0          # [27, 12, 12] structural non-zeros
    assert int(pattern.reshape(27, 4, 3, 4, 3).any(axis=(2, 4)).sum()) == 260
    rng = np.random.default_rng(5)
    Wr = (rng.normal(size=(V, 27, 12, 12)) + 1j * rng.normal(size=(V, 27, 12, 12))) * pattern
    p = B.make_params(pd, B.OK_FP64, storage=fmt)
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wr, torch.complex128), W)
    back = G.unpack_W(p, W, V)
    if fmt == B.OK_W_BLOCK:
        assert np.array_equal(back, Wr)
    else:
        want = Wr.copy()
        for t in range(27):
            ul, ur = Wr[:, t, :6, :6], Wr[:, t, :6, 6:]
            has_ul, has_lr = pattern[t, :6, :6].any(), pattern[t, 6:, 6:].any()
            if has_ul and has_lr:
                want[:, t, 6:, 6:] = ul
            want[:, t, 6:, :6] = -ur if t == 0 else ur
        if fmt == B.OK_W_CONJ:      # W^-_o(x) = [[D^dag, -S^dag], [-S^dag, D^dag]] of W^+_o(x - o), quadrant presence of term t
            for t in range(2, 27, 2):
                src = want[o.sh(np.arange(V), oo.OFFSETS[t]), t - 1]
                D = src[:, :6, :6] if pattern[t - 1, :6, :6].any() else src[:, 6:, 6:]
                Dd, Sd = np.conj(np.swapaxes(D, 1, 2)), np.conj(np.swapaxes(src[:, :6, 6:], 1, 2))
                want[:, t] = 0
                if pattern[t, :6, :6].any():
                    want[:, t, :6, :6] = Dd
                if pattern[t, 6:, 6:].any():
                    want[:, t, 6:, 6:] = Dd
                want[:, t, :6, 6:] = -Sd
                want[:, t, 6:, :6] = -Sd
        assert np.array_equal(back, want)
    psi = I.gaussian_spinor(dims, 3)
    got = G.apply(p, W, psi)
    ref = np.zeros_like(psi)
    for t in range(27):
        ref += np.einsum("nij,nj->ni", back[:, t], psi[o.sh(np.arange(V), oo.OFFSETS[t])])
    assert G.per_site_rel_err(got, ref) <= FP64_TOL


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("case", ["eps", "haar", "periodic"])
def test_sparse_precalc_then_apply(case, prec, fmt):
    dims = (4, 3, 3, 2) if case != "haar" else (4, 4, 4, 8)
    U, pd, o = setup(dims, haar=case == "haar", kappa=0.08 if case == "haar" else 0.10,
                     bc=(1, 1, 1, 1) if case == "periodic" else (1, 1, 1, -1))
    p = B.make_params(pd, prec, storage=fmt)
    W = G.precalc(p, U)
    want_W = o.precalc_W()
    got_W = G.unpack_W(p, W, o.V)
    tolW = 1e-13 if prec == B.OK_FP64 else 2e-7
    assert np.abs(got_W - want_W).max() <= tolW * np.abs(want_W).max()
    assert np.all(got_W[want_W == 0] == 0)
    psi = I.gaussian_spinor(dims, 4)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi, W=want_W)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= FP64_TOL
    else:
        assert G.rel_l2(got, want) <= FP32_TOL
    # a zero field maps to zero, and the padded lanes of the last 32-site block stay zero in the internal layout
    assert np.all(G.apply(p, W, np.zeros_like(psi)) == 0)
    packed_out = B.alloc_vec(p)
    B.ok_dirac_apply(W, G.pack_spinor(p, psi), packed_out)
    torch.cuda.synchronize()
    raw = packed_out.view(torch.float64 if prec == B.OK_FP64 else torch.float32).cpu().numpy()
    nblk = (o.V + 31) // 32
    per = 2 if prec == B.OK_FP64 else 4                       # reals per 16-byte unit
    units = raw.reshape(nblk, -1, 32, per)
    if o.V % 32:
        assert np.all(units[-1, :, o.V % 32:, :] == 0)


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("prec,tol", [(B.OK_FP64, 1e-10), (B.OK_FP32, 1e-6)])
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 3, 3, 2)])            # the second one has a ragged last block (72 sites)
def test_sparse_bicgstab_vs_oracle(dims, prec, tol, fmt):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec, storage=fmt)
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
    assert np.linalg.norm(r) / np.linalg.norm(b) <= tol + (0.0 if prec == B.OK_FP64 else G.fp32_operator_slack(o, xs, b, W=Wc))   # R-RESID
    # bit-reproducible
    x2 = B.alloc_vec(p)
    st2, it2, res2 = B.ok_bicgstab(W, src, x2, tol, 2000, raise_on_fail=False)
    assert (st2, it2, res2) == (st, it, res) and torch.equal(x, x2)
