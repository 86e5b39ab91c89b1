"""Parity of the 12-right-hand-side mode (BASELINE.json configs[3]) with the CPU oracle.

The 12-RHS apply is Eq. (2.2) applied to 12 spinor fields at once: per site a complex
12 x 324 by 324 x 12 contraction on the tensor cores (split fp16, kind::f16).  The oracle side is simply the
single-RHS oracle called column by column.  Tolerance: relative L2 <= 2e-5 per column (north_star, fp32).
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

FP32_TOL = 2e-5
W22_REL = 2.0 ** -22      # split-fp16 W storage: |x - (hi + lo/2048)| <= 2^-11 * 2^-11 |x| (two round-to-nearest fp16 steps)
NR = 12
SHAPES = [(4, 3, 3, 2), (2, 2, 2, 2), (4, 4, 4, 8), (5, 2, 3, 4)]


def setup(dims, eps=0.25, seed=7, kappa=0.10):
    U = I.near_identity_links(dims, eps, seed)
    u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
    pd = I.make_params(dims, kappa, u0)
    return U, pd, Oracle(U, pd)


def gaussian_block(dims, seed0):
    """[V][12 comp][12 rhs]: column j is the seeded Gaussian spinor of seed seed0 + j."""
    return np.stack([I.gaussian_spinor(dims, seed0 + j) for j in range(NR)], axis=2)


def point_sources(dims):
    """All 12 spin-colour point sources at the origin (BASELINE.json configs[3])."""
    return np.stack([I.point_source(dims, site=0, comp=j) for j in range(NR)], axis=2)


def col_rel_l2(got, want):
    num = np.linalg.norm((got - want).reshape(-1, NR), axis=0)
    den = np.linalg.norm(want.reshape(-1, NR), axis=0)
    return float((num / den).max())


@pytest.mark.parametrize("dims", SHAPES)
def test_mrhs_pack_unpack_roundtrip(dims):
    pd = I.make_params(dims, 0.1, 0.95)
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    psi = gaussian_block(dims, 20).astype(np.complex64)
    packed = G.pack_spinor(p, psi)
    assert np.array_equal(G.unpack_spinor(p, packed, psi.shape).astype(np.complex64), psi)
    V = psi.shape[0]
    rng = np.random.default_rng(1)
    Wc = (rng.normal(size=(V, 27, 12, 12)) + 1j * rng.normal(size=(V, 27, 12, 12))).astype(np.complex64)
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wc), W)
    back = G.unpack_W(p, W, V)
    # the 12-RHS W tile stores every real as two fp16 pieces (hi + lo / 2048): 22 significant bits
    err = np.maximum(np.abs(back.real - Wc.real), np.abs(back.imag - Wc.imag))
    ref = np.maximum(np.abs(Wc.real), np.abs(Wc.imag))
    assert np.all(err <= W22_REL * ref + 2.0 ** -36)
    q = B.ok_W_params(W)
    assert list(q.dims) == list(dims) and q.nrhs == NR


@pytest.mark.parametrize("dims", SHAPES)
def test_mrhs_apply_with_oracle_W(dims):
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    Wc = o.precalc_W()
    psi = gaussian_block(dims, 30)
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wc, torch.complex64), W)
    got = G.apply(p, W, psi)
    want = np.stack([o.apply_W(psi[:, :, j], W=Wc) for j in range(NR)], axis=2)
    assert col_rel_l2(got, want) <= FP32_TOL
    # agreement with the single-RHS CUDA path on the same W (both fp32): much tighter than the oracle bound
    p1 = B.make_params(pd, B.OK_FP32)
    W1 = B.alloc_W(p1)
    B.ok_pack_W(p1, G.to_dev(Wc, torch.complex64), W1)
    one = np.stack([G.apply(p1, W1, psi[:, :, j]) for j in range(NR)], axis=2)
    assert col_rel_l2(got, one) <= 5e-6


@pytest.mark.parametrize("dims", SHAPES)
def test_mrhs_precalc_layout_and_apply(dims):
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    W = G.precalc(p, U)
    want_W = o.precalc_W()
    got_W = G.unpack_W(p, W, o.V)
    assert np.abs(got_W - want_W).max() <= (2.0 ** -24 + W22_REL) * np.sqrt(2) * np.abs(want_W).max()
    psi = point_sources(dims)
    got = G.apply(p, W, psi)
    want = np.stack([o.apply_W(psi[:, :, j], W=want_W) for j in range(NR)], axis=2)
    assert col_rel_l2(got, want) <= FP32_TOL
    assert np.all(got[np.abs(want) == 0] == 0)      # exact zeros outside the stencil's support
    assert np.all(G.apply(p, W, np.zeros_like(psi)) == 0)


def run_solver(p, W, b, tol, maxit=2000):
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    st, it, res = B.ok_bicgstab(W, src, x, tol, maxit, raise_on_fail=False)
    return st, it, res, G.unpack_spinor(p, x, b.shape)


@pytest.mark.parametrize("kind", ["point", "gauss"])
def test_mrhs_bicgstab_vs_oracle(kind):
    dims = (4, 4, 4, 8)
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    W = G.precalc(p, U)
    b = point_sources(dims) if kind == "point" else gaussian_block(dims, 40)
    tol = 1e-6
    st, it, res, x = run_solver(p, W, b, tol)
    assert st == 0 and res <= tol
    Wc = o.precalc_W()
    its = []
    for j in range(NR):
        bj = np.ascontiguousarray(b[:, :, j])
        xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), bj, tol, 2000)
        assert sto == 0
        its.append(ito)
        r = bj - o.apply_W(np.ascontiguousarray(x[:, :, j]), W=Wc)
        # R-RESID with the split-fp16 operands of this mode: W and Psi each carry 2^-22 (2 x 4 units of 2^-24 |W||x|) + 1 unit of
        # fp32 accumulation = 9 units against the 2 of the fp32 path
        assert np.linalg.norm(r) / np.linalg.norm(bj) <= tol + 4.5 * G.fp32_operator_slack(o, np.ascontiguousarray(x[:, :, j]), bj, W=Wc)
        assert G.rel_l2(x[:, :, j], xo) <= 20 * tol
    assert abs(it - max(its)) <= 2          # `iters` reports the slowest column


def test_mrhs_bicgstab_edge_cases():
    dims = (4, 4, 4, 8)
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    W = G.precalc(p, U)
    b = gaussian_block(dims, 50)
    b[:, :, 3] = 0                          # one zero column: x_3 = 0, the rest converge
    a1 = run_solver(p, W, b, 1e-6)
    a2 = run_solver(p, W, b, 1e-6)
    assert a1[0] == 0 and a1[2] <= 1e-6 and np.all(a1[3][:, :, 3] == 0)
    assert a1[1] == a2[1] and a1[2] == a2[2] and np.array_equal(a1[3], a2[3])   # bit-reproducible
    st, it, res, x = run_solver(p, W, np.zeros_like(b), 1e-6)
    assert st == 0 and it == 0 and res == 0.0 and np.all(x == 0)
    st, it, res, x = run_solver(p, W, b, 1e-6, maxit=2)
    assert st == -4 and it == 2 and 1e-6 < res < 1.0
