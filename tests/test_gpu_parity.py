"""Parity of the CUDA path (through the C-ABI) with the CPU oracle on identical seeded inputs.

Tolerances (BASELINE.json north_star): fp64 per-site relative error <= 1e-12; fp32 relative L2
error <= 2e-5 (against the fp64 oracle on the same fp64 inputs); BiCGStab iterations within +-2 and
true residual <= tol.  Integer/structural results (zero blocks, padding) are compared exactly.
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
# lattices: ragged tail (72 sites = 2.25 blocks), the 2^4 brute-force lattice (offsets coincide
# modulo L), config 1 (4^3 x 8, 16 blocks), an odd shape with L=2 and L=5
SHAPES = [(4, 3, 3, 2), (2, 2, 2, 2), (4, 4, 4, 8), (5, 2, 3, 4)]


def setup(dims, eps=0.3, seed=1, kappa=0.10, coeffs=None, bc=(1, 1, 1, -1), haar=False):
    U = I.haar_links(dims, seed) if haar else I.near_identity_links(dims, eps, seed)
    u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
    pd = I.make_params(dims, kappa, u0, coeffs=coeffs, bc=bc)
    return U, pd, Oracle(U, pd)


# ------------------------------------------------------------------ layouts
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_pack_unpack_roundtrip(dims, prec):
    pd = I.make_params(dims, 0.1, 0.95)
    p = B.make_params(pd, prec)
    psi = I.gaussian_spinor(dims, 2).astype(G.npdtype(prec))
    packed = G.pack_spinor(p, psi)
    back = G.unpack_spinor(p, packed, psi.shape)
    assert np.array_equal(back.astype(G.npdtype(prec)), psi)
    # padding of the last block is zero
    raw = packed.view(torch.float64 if prec == B.OK_FP64 else torch.float32).cpu().numpy()
    V = psi.shape[0]
    nblk = (V + 31) // 32
    units = raw.reshape(nblk, -1, 32, raw.size // (nblk * 32 * (12 if prec == B.OK_FP64 else 6)))
    if V % 32:
        assert np.all(units[-1, :, V % 32:, :] == 0)
    rng = np.random.default_rng(0)
    Wc = (rng.normal(size=(V, 27, 12, 12)) + 1j * rng.normal(size=(V, 27, 12, 12))).astype(G.npdtype(prec))
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wc), W)
    assert np.array_equal(G.unpack_W(p, W, V).astype(G.npdtype(prec)), Wc)
    q = B.ok_W_params(W)
    assert list(q.dims) == list(dims) and q.precision == prec


# ------------------------------------------------------------------ a3: apply in isolation (oracle W)
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_apply_with_oracle_W(dims, prec):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec)
    Wc = o.precalc_W()
    psi = I.gaussian_spinor(dims, 2)
    W = B.alloc_W(p)
    B.ok_pack_W(p, G.to_dev(Wc, G.cdtype(prec)), W)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi, W=Wc)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= FP64_TOL
    else:
        assert G.rel_l2(got, want) <= FP32_TOL


# ------------------------------------------------------------------ a1+a2: precalc
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_precalc_W_elementwise(dims, prec):
    U, pd, o = setup(dims, eps=0.5, seed=3)
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    got = G.unpack_W(p, W, o.V)
    want = o.precalc_W()
    scale = np.abs(want).max()
    tol = 1e-13 if prec == B.OK_FP64 else 2e-7
    assert np.abs(got - want).max() <= tol * scale
    # structural zeros are exact zeros (P6), 260 non-zero colour blocks
    nz = np.abs(got.reshape(o.V, 27, 4, 3, 4, 3)).max(axis=(0, 3, 5)) > 0
    assert int(nz.sum()) == 260
    assert np.array_equal(nz, np.abs(want.reshape(o.V, 27, 4, 3, 4, 3)).max(axis=(0, 3, 5)) > 1e-14)


@pytest.mark.parametrize("case", ["haar", "periodic", "mixed_bc", "u0_1", "wilson"])
def test_precalc_W_variants(case):
    dims = (4, 3, 2, 4)
    kw = dict(haar=dict(haar=True, kappa=0.08), periodic=dict(bc=(1, 1, 1, 1)), mixed_bc=dict(bc=(-1, 1, -1, -1)),
              u0_1=dict(), wilson=dict(coeffs=I.WILSON))[case]
    U, pd, o = setup(dims, seed=5, **kw)
    if case == "u0_1":
        pd["u0"] = 1.0
        o = Oracle(U, pd)
    p = B.make_params(pd, B.OK_FP64)
    got = G.unpack_W(p, G.precalc(p, U), o.V)
    want = o.precalc_W()
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()


# ------------------------------------------------------------------ full path: links -> W -> M psi
@pytest.mark.parametrize("prec", [B.OK_FP64, B.OK_FP32])
@pytest.mark.parametrize("dims", SHAPES)
def test_precalc_then_apply(dims, prec):
    U, pd, o = setup(dims)
    p = B.make_params(pd, prec)
    W = G.precalc(p, U)
    psi = I.gaussian_spinor(dims, 2)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi)
    if prec == B.OK_FP64:
        assert G.per_site_rel_err(got, want) <= FP64_TOL
        assert G.per_site_rel_err(got, o.apply_direct(psi)) <= FP64_TOL
    else:
        assert G.rel_l2(got, want) <= FP32_TOL


def test_free_field_plane_wave_on_gpu():
    """P2 on the device: U = 1, plane wave with antiperiodic time is an eigenmode (closed form in
    tests/test_oracle_pins.py::free_Mp)."""
    from test_oracle_pins import free_Mp
    dims = (4, 4, 4, 8)
    pd = I.make_params(dims, 0.10, 1.0)
    p = B.make_params(pd, B.OK_FP64)
    W = G.precalc(p, I.unit_links(dims))
    n = (1, 3, 2, 5)
    mom = np.array([2 * np.pi * n[0] / 4, 2 * np.pi * n[1] / 4, 2 * np.pi * n[2] / 4, (2 * n[3] + 1) * np.pi / 8])
    chi = np.array([1.0, -0.5j, 0.25, 2.0 + 1j])
    col = np.array([0.3, 1.0j, -1.2])
    phase = np.exp(1j * (I.site_coords(dims) @ mom))
    psi = phase[:, None] * np.kron(chi, col)[None, :]
    want = phase[:, None] * np.kron(free_Mp(mom, I.OK_LIKE_V1, 0.10) @ chi, col)[None, :]
    assert G.per_site_rel_err(G.apply(p, W, psi), want) <= FP64_TOL


def test_point_source_and_zero_input():
    dims = (4, 4, 4, 8)
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP64)
    W = G.precalc(p, U)
    psi = I.point_source(dims, site=0, comp=0)
    got = G.apply(p, W, psi)
    want = o.apply_W(psi)
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()
    assert np.array_equal(got == 0, np.abs(want) == 0)          # support of the stencil, exactly
    assert np.all(G.apply(p, W, np.zeros_like(psi)) == 0)


# ------------------------------------------------------------------ a4+a5: BiCGStab
def run_solver(p, W, b, tol, maxit=2000):
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    st, it, res = B.ok_bicgstab(W, src, x, tol, maxit, raise_on_fail=False)
    return st, it, res, G.unpack_spinor(p, x, b.shape)


@pytest.mark.parametrize("dims,tol", [((4, 4, 4, 8), 1e-10), ((2, 2, 2, 2), 1e-10), ((4, 3, 3, 2), 1e-12)])
def test_bicgstab_fp64_vs_oracle(dims, tol):
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP64)
    W = G.precalc(p, U)
    b = I.gaussian_spinor(dims, 2)
    st, it, res, x = run_solver(p, W, b, tol)
    Wc = o.precalc_W()
    xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), b, tol, 2000)
    assert st == 0 and sto == 0
    assert abs(it - ito) <= 2
    assert res <= tol
    # true residual recomputed by the oracle from the GPU solution
    r = b - o.apply_W(x, W=Wc)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= tol * 1.0001
    assert abs(np.linalg.norm(r) / np.linalg.norm(b) - res) <= 1e-3 * tol
    assert G.rel_l2(x, xo) <= 50 * tol
    if dims == (2, 2, 2, 2):   # P7 brute force: dense LU
        xs = np.linalg.solve(o.dense_M(), b.reshape(-1)).reshape(b.shape)
        assert G.rel_l2(x, xs) <= 1e-8


def test_bicgstab_fp32_vs_oracle():
    dims = (4, 4, 4, 8)
    U, pd, o = setup(dims, eps=0.25, seed=5)
    p = B.make_params(pd, B.OK_FP32)
    W = G.precalc(p, U)
    b = I.gaussian_spinor(dims, 6)
    tol = 1e-6
    st, it, res, x = run_solver(p, W, b, tol)
    Wc = o.precalc_W()
    xo, ito, reso, sto = oo.bicgstab(lambda v: o.apply_W(v, W=Wc), b, tol, 2000)
    assert st == 0 and abs(it - ito) <= 2 and res <= tol
    # true residual with the fp64 oracle operator on the fp32 solution
    r = b.astype(np.complex64).astype(np.complex128) - o.apply_W(x, W=Wc)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= tol + G.fp32_operator_slack(o, x, b, W=Wc)      # DESIGN.md 10, R-RESID
    assert G.rel_l2(x, xo) <= 20 * tol


def test_bicgstab_is_bit_reproducible_and_handles_edge_cases():
    dims = (4, 4, 4, 8)
    U, pd, o = setup(dims)
    p = B.make_params(pd, B.OK_FP64)
    W = G.precalc(p, U)
    b = I.gaussian_spinor(dims, 2)
    a1 = run_solver(p, W, b, 1e-10)
    a2 = run_solver(p, W, b, 1e-10)
    assert a1[1] == a2[1] and a1[2] == a2[2] and np.array_equal(a1[3], a2[3])
    # zero source -> x = 0, 0 iterations
    st, it, res, x = run_solver(p, W, np.zeros_like(b), 1e-10)
    assert st == 0 and it == 0 and res == 0.0 and np.all(x == 0)
    # maxit reached -> OK_EMAXIT with a valid residual and partial solution
    st, it, res, x = run_solver(p, W, b, 1e-10, maxit=3)
    assert st == -4 and it == 3 and 1e-10 < res < 1.0
    r = b - o.apply_W(x)
    assert abs(np.linalg.norm(r) / np.linalg.norm(b) - res) <= 1e-9


def test_errors_reported_not_crashed():
    dims = (4, 4, 4, 8)
    pd = I.make_params(dims, 0.1, 0.95)
    p = B.make_params(pd, B.OK_FP64)
    junk = B.alloc_bytes(4096)
    junk.zero_()
    v = B.alloc_vec(p)
    with pytest.raises(B.OkError) as e:      # buffer without a W header
        B.ok_dirac_apply(junk, v, B.alloc_vec(p))
    assert e.value.status == -1
    W = G.precalc(p, I.unit_links(dims))
    with pytest.raises(B.OkError):           # out aliases psi
        B.ok_dirac_apply(W, v, v)
    B.ok_set_workspace(None)
    st, it, res = B.ok_bicgstab(W, v, B.alloc_vec(p), 1e-8, 10, raise_on_fail=False)
    assert st == -5
