"""ok_cgnr (CG on M^dag M, PAPER.md:164 / SURVEY.md 8(f) item 4) against oracle.cgnr (pin P9) on identical seeded inputs."""
import numpy as np
import pytest
import torch

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("storage", [B.OK_W_DENSE, B.OK_W_CONJ])
@pytest.mark.parametrize("prec,tol", [(B.OK_FP64, 1e-10), (B.OK_FP32, 1e-6)])
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 3, 3, 2)])
def test_cgnr_vs_oracle(dims, prec, tol, storage):
    U = I.near_identity_links(dims, 0.3, 1)
    pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)))
    o = Oracle(U, pd)
    p = B.make_params(pd, prec, storage=storage)
    W = G.precalc(p, U)
    b = I.gaussian_spinor(dims, 2)
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    st, it, res = B.ok_cgnr(W, src, x, tol, 5000, raise_on_fail=False)
    assert st == 0 and res <= tol
    Wc = o.precalc_W()
    ap = lambda v: o.apply_W(v, W=Wc)
    xo, ito, reso, sto = oo.cgnr(ap, b, tol, 5000)
    assert sto == 0 and abs(it - ito) <= max(2, ito // 50)
    xs = G.unpack_spinor(p, x, b.shape)
    assert np.linalg.norm(b - ap(xs)) / np.linalg.norm(b) <= tol + (0.0 if prec == B.OK_FP64 else G.fp32_operator_slack(o, xs, b, W=Wc))   # R-RESID
    assert G.rel_l2(xs, xo) <= 50 * tol
    x2 = B.alloc_vec(p)
    assert B.ok_cgnr(W, src, x2, tol, 5000, raise_on_fail=False) == (st, it, res) and torch.equal(x, x2)   # bit-reproducible
    st3, it3, res3 = B.ok_cgnr(W, src, x2, tol, 3, raise_on_fail=False)
    assert st3 == -4 and it3 == 3 and res3 > tol
    z = G.pack_spinor(p, np.zeros_like(b))
    assert B.ok_cgnr(W, z, x2, tol, 10, raise_on_fail=False) == (0, 0, 0.0)
