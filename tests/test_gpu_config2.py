"""BASELINE.json configs[1] on the GPU: 8^3 x 16, fp64, links eps = 0.3 seed 3, kappa = 0.10, bc (+,+,+,-).
Gauge covariance under a random SU(3) transform (seed 4) evaluated with the CUDA path alone, element-wise parity of the
apply with the oracle on all 8192 sites, and BiCGStab from a point source at the origin (spin 0, colour 0) to 1e-12
against the oracle's iteration count.  PAPER.md:43-59 (problem statement), 114 (solver)."""
import numpy as np
import pytest

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu
DIMS = (8, 8, 8, 16)


@pytest.fixture(scope="module")
def cfg():
    U = I.near_identity_links(DIMS, 0.3, 3)
    pd = I.make_params(DIMS, 0.10, I.tadpole_u0(I.mean_plaquette(DIMS, U)))
    return U, pd, Oracle(U, pd)


@pytest.mark.parametrize("storage", [B.OK_W_DENSE, B.OK_W_CONJ])
def test_config2_gauge_covariance_on_gpu(cfg, storage):
    U, pd, o = cfg
    g = I.random_gauge_transform(DIMS, 4)
    p = B.make_params(pd, B.OK_FP64, storage=storage)
    psi = I.gaussian_spinor(DIMS, 2)
    W = G.precalc(p, U)
    Wg = G.precalc(p, I.gauge_transform_links(DIMS, U, g))
    lhs = G.apply(p, Wg, I.gauge_transform_spinor(psi, g))          # M[U^g] (g psi)
    rhs = I.gauge_transform_spinor(G.apply(p, W, psi), g)           # g (M[U] psi)
    assert G.per_site_rel_err(lhs, rhs) <= 1e-12


def test_config2_apply_and_point_source_solve(cfg):
    U, pd, o = cfg
    p = B.make_params(pd, B.OK_FP64)
    W = G.precalc(p, U)
    Wc = o.precalc_W()
    psi = I.gaussian_spinor(DIMS, 2)
    assert G.per_site_rel_err(G.apply(p, W, psi), o.apply_W(psi, W=Wc)) <= 1e-12
    b = I.point_source(DIMS, site=0, comp=0)
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    st, it, res = B.ok_bicgstab(W, src, x, 1e-12, 2000, raise_on_fail=False)
    assert st == 0 and res <= 1e-12
    xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), b, 1e-12, 2000)
    assert sto == 0 and abs(it - ito) <= 2
    xs = G.unpack_spinor(p, x, b.shape)
    assert np.linalg.norm(b - o.apply_W(xs, W=Wc)) <= 1e-12                       # ||b|| = 1
    assert G.rel_l2(xs, xo) <= 1e-10
