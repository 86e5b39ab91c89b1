"""Apply parity over awkward lattice shapes, every W storage format and the 12-RHS mode.

Extents 2 and 3 make stencil offsets coincide modulo L (+x and -x, or +2x and -x, hit the same site), odd extents break
the 4-site sector alignment the reduced formats enjoy on production lattices, and most volumes leave a ragged last 32-site
block.  Oracle: Oracle.apply_W (Eq. 2.2) with the oracle's own W; the CUDA side precalculates its W itself.
"""
import numpy as np
import pytest

from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu

SHAPES = [(2, 2, 2, 2), (3, 2, 2, 2), (2, 3, 5, 2), (6, 2, 2, 3), (7, 3, 2, 2), (5, 4, 3, 2), (3, 3, 3, 3), (10, 2, 2, 2),
          (4, 4, 2, 6), (9, 2, 3, 2), (33, 2, 2, 2)]
FORMATS = [B.OK_W_DENSE, B.OK_W_BLOCK, B.OK_W_DS, B.OK_W_CONJ]


@pytest.fixture(scope="module")
def cases():
    out = {}
    for k, dims in enumerate(SHAPES):
        U = I.near_identity_links(dims, 0.3, 100 + k)
        pd = I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U)), bc=(1, 1, 1, -1) if k % 3 else (-1, 1, -1, -1))
        o = Oracle(U, pd)
        psi = I.gaussian_spinor(dims, 200 + k)
        out[dims] = (U, pd, o, psi, o.apply_W(psi))
    return out


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_apply_all_formats_all_shapes(cases, dims, prec, fmt):
    U, pd, o, psi, want = cases[dims]
    p = B.make_params(pd, prec, storage=fmt)
    W = G.precalc(p, U)
    got = G.apply(p, W, psi)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= 1e-12
    else:
        assert G.rel_l2(got, want) <= 2e-5


@pytest.mark.parametrize("dims", SHAPES)
def test_apply_12rhs_all_shapes(cases, dims):
    U, pd, o, psi, want = cases[dims]
    p = B.make_params(pd, B.OK_FP32, nrhs=12)
    W = G.precalc(p, U)
    block = np.stack([np.roll(psi, 7 * j, axis=0) * (10.0 ** (j - 6)) for j in range(12)], axis=2)   # columns of very different scale
    got = G.apply(p, W, block)
    ref = o.apply_W(block)
    num = np.linalg.norm((got - ref).reshape(-1, 12), axis=0)
    den = np.linalg.norm(ref.reshape(-1, 12), axis=0)
    assert float((num / den).max()) <= 2e-5
