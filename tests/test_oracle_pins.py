"""Pins of the CPU oracle against what the paper and the mathematics fix.

Nothing here compares the oracle with itself through the same formula: each pin is either a
second independent evaluation (direct gauge-link form, hand-coded textbook operator written
with np.roll on the 4-d array instead of the oracle's index tables), a closed form, an
invariance, or brute force.
"""
import json
import os

import numpy as np
import pytest

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle, OFFSETS, GAMMA, GAMMA5, SIGMA
from paper_1311_5029_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


# ----------------------------------------------------------------------------- paper facts
def test_paper_structural_facts():
    """27 terms; 27 x 16 = 432 colour blocks; temporal reach 1, spatial reach 2."""
    facts = json.load(open(os.path.join(GOLD, "paper_facts.json")))
    assert OFFSETS.shape == (facts["stencil_terms"], 4)
    assert OFFSETS.shape[0] * 16 == facts["colour_blocks_full_W"]
    assert len({tuple(o) for o in OFFSETS}) == 27
    assert np.abs(OFFSETS[:, 3]).max() == facts["temporal_reach"]
    assert np.abs(OFFSETS[:, :3]).sum(axis=1).max() == facts["spatial_reach"]
    # every offset's opposite is in the table (conjugate pairs)
    S = {tuple(o) for o in OFFSETS}
    assert all(tuple(-o) in S for o in OFFSETS)
    # terms with a temporal hop have no spatial hop
    assert all(np.abs(o[:3]).sum() == 0 for o in OFFSETS if o[3] != 0)


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("dims,u0,eps", [((4, 3, 3, 2), 1.0, 0.6), ((4, 3, 3, 2), 0.93, 0.6),
                                         ((2, 2, 2, 2), 0.9, 0.8), ((3, 2, 4, 5), 0.95, 0.4)])
def test_P1_direct_equals_W_form(dims, u0, eps):
    U = I.near_identity_links(dims, eps, seed=11)
    o = Oracle(U, I.make_params(dims, 0.10, u0))
    psi = I.gaussian_spinor(dims, 5)
    assert rel(o.apply_W(psi), o.apply_direct(psi)) < 1e-13


def test_P1_direct_equals_W_form_haar_and_periodic():
    dims = (4, 3, 3, 2)
    U = I.haar_links(dims, 3)
    psi = I.gaussian_spinor(dims, 5)
    for bc in [(1, 1, 1, -1), (1, 1, 1, 1), (-1, 1, -1, -1)]:
        o = Oracle(U, I.make_params(dims, 0.08, 0.9, bc=bc))
        assert rel(o.apply_W(psi), o.apply_direct(psi)) < 1e-13


def test_P1_each_coefficient_alone():
    """One coefficient at a time, so a compensating pair of mistakes cannot hide."""
    dims = (3, 3, 2, 2)
    U = I.near_identity_links(dims, 0.7, 13)
    psi = I.gaussian_spinor(dims, 6)
    for name in ["cB", "cE", "cEE", "c1", "c2", "c3", "c4", "c5"]:
        c = dict(I.WILSON)
        c[name] = 0.37
        o = Oracle(U, I.make_params(dims, 0.11, 0.91, coeffs=c))
        assert rel(o.apply_W(psi), o.apply_direct(psi)) < 1e-13, name


# ----------------------------------------------------------------------------- P2 free field
def free_Mp(p, c, kappa):
    """Closed form M(p) for U = 1, u0 = 1, derived by hand from Eqs. (2.6)-(2.12) (P2)."""
    g = GAMMA
    M = (1 / (2 * kappa) - np.cos(p[3])) * np.eye(4) + 1j * g[3] * np.sin(p[3])
    for i in range(3):
        M = M + (-(c["rs"] * c["zeta"] + 8 * c["c4"]) * np.cos(p[i]) + 2 * c["c4"] * np.cos(2 * p[i])) * np.eye(4)
        others = sum(np.cos(p[j]) for j in range(3) if j != i)
        M = M + 1j * g[i] * ((c["zeta"] - 2 * c["c1"] - 12 * c["c2"]) * np.sin(p[i])
                             + (c["c1"] + 2 * c["c2"]) * np.sin(2 * p[i]) + 4 * c["c2"] * np.sin(p[i]) * others)
    return M


def test_P2_free_field_W_closed_forms():
    dims = (4, 4, 3, 4)
    c = I.OK_LIKE_V1
    kappa = 0.10
    o = Oracle(I.unit_links(dims), I.make_params(dims, kappa, 1.0, bc=(1, 1, 1, 1)))
    W = o.precalc_W(np.array([0, 7, 50]))
    one = np.eye(3)
    g = GAMMA
    exp = [np.eye(4) / (2 * kappa)]
    a, b = -0.5 * (c["rs"] * c["zeta"] + 8 * c["c4"]), 0.5 * (c["zeta"] - 2 * c["c1"] - 12 * c["c2"])
    for i in range(3):
        exp += [a * np.eye(4) + b * g[i], a * np.eye(4) - b * g[i]]
    exp += [-0.5 * (np.eye(4) - g[3]), -0.5 * (np.eye(4) + g[3])]
    for i in range(3):
        exp += [c["c4"] * np.eye(4) + 0.5 * (c["c1"] + 2 * c["c2"]) * g[i],
                c["c4"] * np.eye(4) - 0.5 * (c["c1"] + 2 * c["c2"]) * g[i]]
    for i, j in [(0, 1), (0, 2), (1, 2)]:
        exp += [c["c2"] * (g[i] + g[j]), -c["c2"] * (g[i] + g[j]), c["c2"] * (g[i] - g[j]), -c["c2"] * (g[i] - g[j])]
    for t in range(27):
        for s in range(3):
            assert np.abs(W[s, t] - np.kron(exp[t], one)).max() < 1e-14, t


@pytest.mark.parametrize("n", [(1, 0, 2, 1), (0, 0, 0, 0), (3, 2, 1, 3)])
def test_P2_plane_wave_is_eigenmode(n):
    """psi = e^{ipx} chi (x) c with p_i = 2 pi n_i/L_i, p_4 = (2 n_4 + 1) pi / T (antiperiodic)."""
    dims = (4, 4, 3, 6)
    c = I.OK_LIKE_V1
    kappa = 0.10
    o = Oracle(I.unit_links(dims), I.make_params(dims, kappa, 1.0))
    p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1], 2 * np.pi * n[2] / dims[2],
                  (2 * n[3] + 1) * np.pi / dims[3]])
    rng = np.random.default_rng(0)
    chi = rng.normal(size=4) + 1j * rng.normal(size=4)
    col = rng.normal(size=3) + 1j * rng.normal(size=3)
    phase = np.exp(1j * (I.site_coords(dims) @ p))
    psi = phase[:, None] * np.kron(chi, col)[None, :]
    want = phase[:, None] * np.kron(free_Mp(p, c, kappa) @ chi, col)[None, :]
    assert rel(o.apply_W(psi), want) < 1e-13
    assert rel(o.apply_direct(psi), want) < 1e-13


def test_P2_continuum_limit():
    """Independent of Eqs. (2.6)-(2.12): the improvement terms are O(p^3), so for small p
    M(p) = m0 + i g4 p4 + p4^2/2 + i zeta g.p + rs zeta p^2/2 + O(p^3),
    m0 = 1/(2 kappa) - (1 + 3 rs zeta + 18 c4).  M(p) is assembled from the oracle's
    free-field W matrices as sum_o W_o e^{i p.o}."""
    dims = (4, 4, 4, 4)
    c = I.OK_LIKE_V1
    kappa = 0.10
    o = Oracle(I.unit_links(dims), I.make_params(dims, kappa, 1.0, bc=(1, 1, 1, 1)))
    W = o.precalc_W(np.array([0]))[0]
    p = 1e-3 * np.array([0.7, -1.1, 0.4, 0.9])
    Mp = sum(W[t] * np.exp(1j * (OFFSETS[t] @ p)) for t in range(27))
    m0 = 1 / (2 * kappa) - (1 + 3 * c["rs"] * c["zeta"] + 18 * c["c4"])
    want = (m0 + 0.5 * p[3] ** 2 + 0.5 * c["rs"] * c["zeta"] * (p[:3] @ p[:3])) * np.eye(4) + 1j * GAMMA[3] * p[3]
    want = want + 1j * c["zeta"] * sum(GAMMA[i] * p[i] for i in range(3))
    assert np.abs(Mp - np.kron(want, np.eye(3))).max() < 20 * np.abs(p).max() ** 3


# ----------------------------------------------------------------------------- P3
def test_P3_gauge_covariance():
    dims = (4, 3, 2, 4)
    U = I.near_identity_links(dims, 0.5, 21)
    p = I.make_params(dims, 0.10, 0.94)
    g = I.random_gauge_transform(dims, 4)
    psi = I.gaussian_spinor(dims, 7)
    o, og = Oracle(U, p), Oracle(I.gauge_transform_links(dims, U, g), p)
    lhs = og.apply_W(I.gauge_transform_spinor(psi, g))
    rhs = I.gauge_transform_spinor(o.apply_W(psi), g)
    assert rel(lhs, rhs) < 1e-13
    # per term: W'_o(x) = g(x) W_o(x) g(x+o)^dag (colour only)
    idx = np.arange(o.V)
    W, Wg = o.precalc_W(idx), og.precalc_W(idx)
    for t in range(27):
        gx = np.einsum("st,nab->nsatb", np.eye(4), g).reshape(-1, 12, 12)
        gy = np.einsum("st,nab->nsatb", np.eye(4), g[o.sh(idx, OFFSETS[t])]).reshape(-1, 12, 12)
        assert rel(Wg[:, t], gx @ W[:, t] @ oo.dag(gy)) < 1e-12, t


# ----------------------------------------------------------------------------- P4
def test_P4_gamma5_hermiticity_dense_2p4():
    dims = (2, 2, 2, 2)
    U = I.near_identity_links(dims, 0.5, 31)
    o = Oracle(U, I.make_params(dims, 0.10, 0.95))
    M = o.dense_M()
    G5 = np.kron(np.eye(o.V), np.kron(GAMMA5, np.eye(3)))
    assert np.abs(G5 @ M @ G5 - M.conj().T).max() / np.abs(M).max() < 1e-14


def test_P4_gamma5_hermiticity_inner_product():
    dims = (4, 3, 3, 4)
    U = I.near_identity_links(dims, 0.4, 32)
    o = Oracle(U, I.make_params(dims, 0.10, 0.95))
    phi, psi = I.gaussian_spinor(dims, 8), I.gaussian_spinor(dims, 9)
    g5 = np.kron(GAMMA5, np.eye(3))
    lhs = np.vdot(phi, o.apply_W(psi))
    rhs = np.vdot((o.apply_W(phi @ g5.T)) @ g5.T, psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


def test_conjugation_relations_2_3_and_2_12():
    """Eq. (2.3): W^{+-}_{ji,x} built through the relation equals Eq. (2.12)
    evaluated directly with i <-> j (a second route to the same matrix)."""
    dims = (3, 4, 3, 2)
    U = I.near_identity_links(dims, 0.6, 33)
    o = Oracle(U, I.make_params(dims, 0.10, 0.9))
    idx = np.arange(o.V)
    W = o.precalc_W(idx)
    for q, (i, j) in enumerate(oo.PAIRS):
        S = o.S_pm_ij(j, i, idx)               # (2.12) with the roles of i and j exchanged
        Z = np.zeros_like(S)
        assert rel(W[:, 18 + 4 * q], oo.blocks(Z, S, S, Z)) < 1e-13


# ----------------------------------------------------------------------------- P5 textbook operators
def _roll(f, dims, mu, s, bc=1):
    """f(x + s*mu_hat) on the 4-d array, with the boundary sign for fermion fields."""
    Lx, Ly, Lz, T = dims
    a = f.reshape((T, Lz, Ly, Lx) + f.shape[1:])
    ax = 3 - mu
    r = np.roll(a, -s, axis=ax).copy()
    if bc == -1:
        sl = [slice(None)] * 4
        sl[ax] = slice(-1, None) if s == 1 else slice(0, 1)
        r[tuple(sl)] *= -1
    return r.reshape(f.shape)


def wilson_apply(dims, U, kappa, psi, bc):
    """Textbook Wilson operator, hand-coded:
    M psi = psi/(2k) - 1/2 sum_mu [(1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu(x-mu)^dag psi(x-mu)]."""
    V = psi.shape[0]
    f = psi.reshape(V, 4, 3)
    out = f / (2 * kappa)
    for mu in range(4):
        fwd = np.einsum("nab,nsb->nsa", U[:, mu], _roll(f, dims, mu, +1, bc[mu]))
        Ub = _roll(U[:, mu], dims, mu, -1)
        bwd = np.einsum("nba,nsb->nsa", Ub.conj(), _roll(f, dims, mu, -1, bc[mu]))
        out = out - 0.5 * (np.einsum("st,ntc->nsc", np.eye(4) - GAMMA[mu], fwd)
                           + np.einsum("st,ntc->nsc", np.eye(4) + GAMMA[mu], bwd))
    return out.reshape(V, 12)


def clover_F(dims, U, mu, nu):
    """Hand-coded clover F_mu,nu with np.roll (independent of Oracle.F's index tables)."""
    R = lambda A, d, s: _roll(A, dims, d, s)
    d = lambda A: np.conj(np.swapaxes(A, -1, -2))
    Um, Un = U[:, mu], U[:, nu]
    Q = Um @ R(Un, mu, 1) @ d(R(Um, nu, 1)) @ d(Un)
    Q = Q + Un @ d(R(R(Um, mu, -1), nu, 1)) @ d(R(Un, mu, -1)) @ R(Um, mu, -1)
    Q = Q + d(R(Um, mu, -1)) @ d(R(R(Un, mu, -1), nu, -1)) @ R(R(Um, mu, -1), nu, -1) @ R(Un, nu, -1)
    Q = Q + d(R(Un, nu, -1)) @ R(Um, nu, -1) @ R(R(Un, mu, 1), nu, -1) @ d(Um)
    return (Q - d(Q)) / 8


@pytest.mark.parametrize("bc", [(1, 1, 1, -1), (1, 1, 1, 1)])
def test_P5_wilson_special_case(bc):
    dims = (4, 3, 2, 4)
    U = I.near_identity_links(dims, 0.5, 41)
    psi = I.gaussian_spinor(dims, 10)
    o = Oracle(U, I.make_params(dims, 0.12, 1.0, coeffs=I.WILSON, bc=bc))
    want = wilson_apply(dims, U, 0.12, psi, bc)
    assert rel(o.apply_W(psi), want) < 1e-13
    assert rel(o.apply_direct(psi), want) < 1e-13


def test_P5_wilson_clover_special_case():
    """cB = cE = c_SW: M = Wilson + (i/4) c_SW sum_{mu,nu} sigma_mu,nu F_mu,nu with
    sigma_mu,nu = (i/2)[g_mu, g_nu] and the anti-Hermitian clover F (hypercubic scalar)."""
    dims = (4, 3, 2, 4)
    bc = (1, 1, 1, -1)
    csw = 1.3
    U = I.near_identity_links(dims, 0.5, 42)
    psi = I.gaussian_spinor(dims, 11)
    c = dict(I.WILSON)
    c["cB"] = c["cE"] = csw
    o = Oracle(U, I.make_params(dims, 0.12, 1.0, coeffs=c, bc=bc))
    V = psi.shape[0]
    f = psi.reshape(V, 4, 3)
    clov = np.zeros_like(f)
    for mu in range(4):
        for nu in range(4):
            if mu != nu:
                sig = 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
                clov = clov + np.einsum("st,nab,ntb->nsa", sig, clover_F(dims, U, mu, nu), f)
    want = wilson_apply(dims, U, 0.12, psi, bc) + (0.25j * csw * clov).reshape(V, 12)
    assert rel(o.apply_W(psi), want) < 1e-13


def test_field_strength_properties():
    """F anti-Hermitian, F_mu,nu = -F_nu,mu, unchanged by the boundary fold, zero on pure gauge."""
    dims = (3, 3, 2, 4)
    U = I.near_identity_links(dims, 0.6, 43)
    o = Oracle(U, I.make_params(dims, 0.1, 1.0))
    op = Oracle(U, I.make_params(dims, 0.1, 1.0, bc=(1, 1, 1, 1)))
    idx = np.arange(o.V)
    for mu in range(4):
        for nu in range(mu + 1, 4):
            F = o.F(mu, nu, idx)
            assert np.abs(F + oo.dag(F)).max() < 1e-15
            assert np.abs(F + o.F(nu, mu, idx)).max() < 1e-15
            assert np.abs(F - op.F(mu, nu, idx)).max() == 0.0
            assert rel(F, clover_F(dims, U, mu, nu)) < 1e-14
    g = I.random_gauge_transform(dims, 5)
    pure = Oracle(I.gauge_transform_links(dims, I.unit_links(dims), g), I.make_params(dims, 0.1, 1.0))
    assert np.abs(pure.F(0, 3, idx)).max() < 1e-14
    # weak-field limit: a constant abelian-like field U_mu = exp(i a_mu(x)) in the lambda_3 direction
    # with a_y = b*x gives plaquette exp(i b): F_xy = i sin(b) lambda_3-direction generator (periodic
    # seam excluded) -- fixes the 1/8 normalisation and the orientation of Q.
    dims2 = (6, 4, 2, 2)
    b = 0.05
    T3 = np.diag([1.0, -1.0, 0.0])
    Ua = I.unit_links(dims2)
    x = I.site_coords(dims2)[:, 0]
    Ua[:, 1] = np.einsum("n,ij->nij", np.exp(1j * b * x), np.diag([1.0, 0, 0])) \
        + np.einsum("n,ij->nij", np.exp(-1j * b * x), np.diag([0, 1.0, 0])) + np.diag([0, 0, 1.0])[None]
    oa = Oracle(Ua, I.make_params(dims2, 0.1, 1.0, bc=(1, 1, 1, 1)))
    interior = np.where((x >= 1) & (x <= dims2[0] - 2))[0]
    Fxy = oa.F(0, 1, interior)
    assert np.abs(Fxy - 1j * np.sin(b) * T3[None]).max() < 1e-14


# ----------------------------------------------------------------------------- P6 structure
def test_P6_zero_block_structure():
    dims = (3, 3, 3, 2)
    U = I.haar_links(dims, 51)
    o = Oracle(U, I.make_params(dims, 0.08, 0.9))
    W = o.precalc_W(np.arange(6))
    nz = []
    for t in range(27):
        blk = np.abs(W[:, t].reshape(6, 4, 3, 4, 3)).max(axis=(0, 2, 4)) > 1e-14      # [alpha, beta]
        nz.append(int(blk.sum()))
    want = [16] + [16] * 6 + [10, 10] + [8] * 6 + [4] * 4 + [8] * 8
    assert nz == want
    assert sum(nz) == 260
    # block forms of Eqs. (2.6)-(2.12): W^+_i, W^++_ii = [[D,S],[S,D]]; W^0 - mass = [[D,S],[-S,D]]
    for t in [1, 3, 5, 9, 11, 13]:
        assert np.abs(W[:, t, :6, :6] - W[:, t, 6:, 6:]).max() == 0 and np.abs(W[:, t, :6, 6:] - W[:, t, 6:, :6]).max() == 0
    assert np.abs(W[:, 0, :6, 6:] + W[:, 0, 6:, :6]).max() == 0
    assert np.abs(W[:, 7, :6, :6]).max() == 0 and np.abs(W[:, 8, 6:, 6:]).max() == 0


def test_staple_content_of_c5_hop_term():
    """Eq. (2.8)'s (c5/4)(u0^-2 - u0^-4) term: the products B U in the last bracket of
    D^+_i contain 3-link staples (a clover leaf ending in U_i^dag(x) times U_i(x)).  Their sum must be
    (i/4) sum_jk eps_ijk sigma_j (staple_up_k - staple_down_k).  Extract it as the part of the bracket
    that is invariant under U_i(x0) -> e^{i theta} U_i(x0) on one link (5-link terms carry e^{+-i theta})."""
    dims = (4, 4, 4, 2)
    U = I.near_identity_links(dims, 0.7, 61)
    c = dict(I.WILSON)
    c["rs"] = 0.0
    c["c5"] = 1.0
    x0 = 21
    for i in range(3):
        acc = 0
        nth = 8
        for th in range(nth):
            Ut = U.copy()
            Ut[x0, i] *= np.exp(2j * np.pi * th / nth)
            o = Oracle(Ut, I.make_params(dims, 0.1, 1.0, coeffs=c, bc=(1, 1, 1, 1)))
            D, _ = o.DS_plus(i, np.array([x0]))
            acc = acc + D[0] / nth
        o = Oracle(U, I.make_params(dims, 0.1, 1.0, coeffs=c, bc=(1, 1, 1, 1)))
        want = np.zeros((6, 6), dtype=complex)
        for j in range(3):
            for k in range(3):
                if oo.EPS[i, j, k]:
                    G = o.staple_up(i, k, np.array([x0])) - o.staple_down(i, k, np.array([x0]))
                    want += 0.25j * oo.EPS[i, j, k] * np.kron(SIGMA[j], G[0])
        assert np.abs(acc - want).max() < 1e-14


# ----------------------------------------------------------------------------- P7 solver
def test_P7_bicgstab_vs_dense_LU_2p4():
    dims = (2, 2, 2, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    plaq = I.mean_plaquette(dims, U)
    o = Oracle(U, I.make_params(dims, 0.10, I.tadpole_u0(plaq)))
    M = o.dense_M()
    b = I.gaussian_spinor(dims, 2)
    W = o.precalc_W()
    x, it, res, st = oo.bicgstab(lambda v: o.apply_W(v, W=W), b, 1e-10, 500)
    xs = np.linalg.solve(M, b.reshape(-1)).reshape(b.shape)
    assert st == 0 and res <= 1e-10
    assert rel(x, xs) < 1e-9


def test_bicgstab_textbook_small_matrix():
    """The solver routine on a generic well-conditioned complex matrix vs numpy's LU."""
    rng = np.random.default_rng(3)
    n = 60
    A = 4 * np.eye(n) + 0.3 * (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    x, it, res, st = oo.bicgstab(lambda v: A @ v, b, 1e-12, 200)
    assert st == 0 and res <= 1e-12 and it < 60
    assert rel(x, np.linalg.solve(A, b)) < 1e-10
    # exact-arithmetic property: at most n iterations; breakdown code on a singular start
    x, it, res, st = oo.bicgstab(lambda v: 0 * v, b, 1e-12, 5)
    assert st == -3


# ----------------------------------------------------------------------------- P8 mixed-precision inversion (R-MIXED)
def test_P8_mixed_precision_vs_dense_LU_2p4():
    """Defect correction around a complex64 BiCGStab reaches the fp64 solution of the dense matrix (LU), the inner
    solver alone cannot; the number of outer corrections follows from the contraction factor inner_tol per correction."""
    dims = (2, 2, 2, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    o = Oracle(U, I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U))))
    M = o.dense_M()
    b = I.gaussian_spinor(dims, 2)
    W = o.precalc_W()
    W32 = W.astype(np.complex64)
    hi = lambda v: o.apply_W(v, W=W)
    lo = lambda v: np.einsum("ntij,tnj->ni", W32, np.stack([v[o.sh(np.arange(o.V), off)] for off in oo.OFFSETS])).astype(np.complex64)
    xs = np.linalg.solve(M, b.reshape(-1)).reshape(b.shape)
    x, its, outer, res, st = oo.bicgstab_mixed(hi, lo, b, 1e-12, 1e-4, 1000)
    assert st == 0 and res <= 1e-12 and rel(x, xs) < 1e-11
    assert 3 <= outer <= 5                       # 1e-12 at 1e-4 (or better) per correction
    # the low-precision inverter on its own stalls at single-precision level
    x32, it32, res32, st32 = oo.bicgstab(lo, b.astype(np.complex64), 1e-12, 300)
    assert rel(x32.astype(np.complex128), xs) > 1e-8
    # exact low-precision operator (lo == hi): one correction of accuracy inner_tol per outer step
    x, its, outer, res, st = oo.bicgstab_mixed(hi, hi, b, 1e-9, 1e-3, 1000, lo_dtype=np.complex128)
    assert st == 0 and outer == 3 and rel(x, xs) < 1e-8
    # zero right-hand side, and the iteration budget
    x, its, outer, res, st = oo.bicgstab_mixed(hi, lo, 0 * b, 1e-12, 1e-4, 1000)
    assert st == 0 and its == 0 and outer == 0 and np.all(x == 0)
    x, its, outer, res, st = oo.bicgstab_mixed(hi, lo, b, 1e-12, 1e-4, 5)
    assert st == -4 and its == 5 and res > 1e-12


# ----------------------------------------------------------------------------- P9 CG on the normal equations
def test_P9_cgnr_vs_dense_LU_and_gamma5():
    dims = (2, 2, 2, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    o = Oracle(U, I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U))))
    M = o.dense_M()
    W = o.precalc_W()
    ap = lambda v: o.apply_W(v, W=W)
    b = I.gaussian_spinor(dims, 2)
    # Gamma_5 M Gamma_5 is the adjoint of the dense matrix, so CGNR's M^dag is the true one
    v = I.gaussian_spinor(dims, 5)
    want = (M.conj().T @ v.reshape(-1)).reshape(v.shape)
    assert rel(oo.gamma5_mul(ap(oo.gamma5_mul(v))), want) < 1e-13
    assert rel(oo.gamma5_mul(oo.gamma5_mul(v)), v) < 1e-15                      # gamma_5^2 = 1
    x, it, res, st = oo.cgnr(ap, b, 1e-10, 2000)
    xs = np.linalg.solve(M, b.reshape(-1)).reshape(b.shape)
    assert st == 0 and res <= 1e-10 and rel(x, xs) < 1e-8
    assert it <= 192                                                          # exact arithmetic: at most dim(M) steps
    # textbook property: the residual norm of M^dag M x = M^dag b decreases monotonically in the M^dag M energy norm;
    # here we check the cheap consequence that CGNR never needs more M applies than 2 x dim on a well-conditioned matrix
    rng = np.random.default_rng(4)
    x0, it0, res0, st0 = oo.cgnr(ap, 0 * b, 1e-10, 10)
    assert st0 == 0 and it0 == 0 and np.all(x0 == 0)
    x1, it1, res1, st1 = oo.cgnr(ap, b, 1e-10, 3)
    assert st1 == -4 and it1 == 3 and res1 > 1e-10


# ---------------------------------------------------------------------------------------------------------------
# P10: cubic-group covariance.  The OK action is built from lattice-covariant objects (an improved
# Wilson-type action; Eqs. 2.6-2.12 treat the three spatial directions alike), so a rotation of the gauge field by 90
# degrees about a spatial axis, with the spinor rotated by the matching S, must commute with M; likewise spatial parity
# with psi -> gamma_4 psi.  This pins what P1-P9 cannot: the assignment of sigma_i to direction i, the orientation of
# B_i = eps_ijk F_jk / 2 against the links it multiplies, and the placement of the E (vector) and B (axial) terms in the
# off-diagonal / diagonal spin blocks -- a plausible slip there (a swapped pair of B components, a wrong sign on one of
# them, E in a diagonal block) leaves every earlier pin green if made consistently in both evaluations of the operator.
def _coords(dims):
    return I.site_coords(dims)


def _index(dims, c):
    Lx, Ly, Lz, T = dims
    return c[:, 0] + Lx * (c[:, 1] + Ly * (c[:, 2] + Lz * c[:, 3]))


def _rotated_links(dims, U, a, b):
    """Image of the gauge field under the rotation by +90 degrees in the (a, b) plane: direction a -> b, b -> -a
    (L_a = L_b).  The link x -> x + a becomes the link x' -> x' + b; the link x -> x + b becomes x' -> x' - a, i.e.
    the reversed link U'_a(x' - a); all other links keep their direction."""
    c = _coords(dims)
    cp = c.copy()
    cp[:, a] = (-c[:, b]) % dims[a]
    cp[:, b] = c[:, a]
    img = _index(dims, cp)                      # img[n] = index of R x_n
    Up = np.empty_like(U)
    Up[img, b] = U[:, a]
    cm = cp.copy()
    cm[:, a] = (cm[:, a] - 1) % dims[a]
    Up[_index(dims, cm), a] = oo.dag(U[:, b])
    for mu in range(4):
        if mu not in (a, b):
            Up[img, mu] = U[:, mu]
    return Up, img


@pytest.mark.parametrize("plane", [(0, 1), (1, 2), (2, 0)])
def test_P10_rotation_covariance(plane):
    a, b = plane
    dims = [3, 3, 3, 2]
    dims[a] = dims[b] = 4
    dims = tuple(dims)
    U = I.near_identity_links(dims, 0.4, 21)
    pd = I.make_params(dims, 0.11, 0.93)
    Up, img = _rotated_links(dims, U, a, b)
    # the spinor representation is DEFINED by S gamma_mu S^-1 = gamma_(R mu): R a = b, R b = -a
    S = (np.eye(4) - GAMMA[a] @ GAMMA[b]) / np.sqrt(2.0)
    Si = np.linalg.inv(S)
    assert np.allclose(S @ GAMMA[a] @ Si, GAMMA[b]) and np.allclose(S @ GAMMA[b] @ Si, -GAMMA[a])
    for mu in range(4):
        if mu not in (a, b):
            assert np.allclose(S @ GAMMA[mu] @ Si, GAMMA[mu])
    psi = I.gaussian_spinor(dims, 22)
    V = psi.shape[0]

    def rot(f):                                 # (T f)(R x) = S f(x)
        g = np.empty_like(f)
        g[img] = np.einsum("st,ntc->nsc", S, f.reshape(V, 4, 3)).reshape(V, 12)
        return g

    lhs = Oracle(Up, pd).apply_W(rot(psi))
    rhs = rot(Oracle(U, pd).apply_W(psi))
    assert np.linalg.norm(lhs - rhs) <= 1e-12 * np.linalg.norm(rhs)
    # the direct (link-product) evaluation obeys it too
    lhs_d = Oracle(Up, pd).apply_direct(rot(psi))
    assert np.linalg.norm(lhs_d - rhs) <= 1e-12 * np.linalg.norm(rhs)
    # and the check has teeth: the unrotated spinor map fails
    g = np.empty_like(psi)
    g[img] = psi
    assert np.linalg.norm(Oracle(Up, pd).apply_W(g) - rhs) > 1e-2 * np.linalg.norm(rhs)


def test_P10_spatial_parity_covariance():
    dims = (4, 3, 3, 2)
    U = I.near_identity_links(dims, 0.4, 23)
    pd = I.make_params(dims, 0.11, 0.93)
    c = _coords(dims)
    cp = c.copy()
    for i in range(3):
        cp[:, i] = (-c[:, i]) % dims[i]
    img = _index(dims, cp)
    Up = np.empty_like(U)
    for i in range(3):                          # the link x -> x + i becomes x' -> x' - i: the reversed link U'_i(x' - i)
        cm = cp.copy()
        cm[:, i] = (cm[:, i] - 1) % dims[i]
        Up[_index(dims, cm), i] = oo.dag(U[:, i])
    Up[img, 3] = U[:, 3]
    psi = I.gaussian_spinor(dims, 24)
    V = psi.shape[0]

    def par(f):                                 # (P f)(-x, t) = gamma_4 f(x, t); gamma_4 gamma_i gamma_4 = -gamma_i
        g = np.empty_like(f)
        g[img] = np.einsum("st,ntc->nsc", GAMMA[3], f.reshape(V, 4, 3)).reshape(V, 12)
        return g

    lhs = Oracle(Up, pd).apply_W(par(psi))
    rhs = par(Oracle(U, pd).apply_W(psi))
    assert np.linalg.norm(lhs - rhs) <= 1e-12 * np.linalg.norm(rhs)
    g = np.empty_like(psi)
    g[img] = psi                                # without gamma_4 the E terms and the hops come out with the wrong sign
    assert np.linalg.norm(Oracle(Up, pd).apply_W(g) - rhs) > 1e-2 * np.linalg.norm(rhs)
