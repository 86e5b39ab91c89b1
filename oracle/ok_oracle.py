"""CPU ORACLE for the Oktay-Kronfeld (OK) action hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Plain numpy, fp64, written from /root/reference/PAPER.md (arXiv:1311.5029) and the readings
listed in DESIGN.md ("Readings of the paper").  It shares no code with the CUDA path
(paper_1311_5029_b200/csrc, binding.py) and imports nothing from it.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it.

What it computes, and the passage each function follows:

  fold_bc            antiperiodic-time sign folded into the links          DESIGN.md R-BC
  field_strength     clover F_mu,nu ; E_i = F_4i ; B_i = eps_ijk F_jk / 2   DESIGN.md R-F (PAPER.md:91 names E,B only)
  precalc_W          the 27 "precalculation matrices" W of Eq. (2.2)        PAPER.md:89-107, Eqs. (2.6)-(2.12), (2.3), (2.10)
  apply_W            sum_y M_xy psi_y in collected form                     PAPER.md:53-55, Eq. (2.2)
  apply_direct       the same operator as raw gauge-link products           DESIGN.md R-DIRECT (the paper's "Naive")
  bicgstab           bi-stabilised CG, textbook van der Vorst               PAPER.md:114 ; DESIGN.md R-SOLVER
  bicgstab_mixed     mixed-precision inversion: defect correction around    PAPER.md:114 ("mixed precision inversion by calling
                     a low-precision bicgstab                               the inverter ... in single or double precision") ; R-MIXED
  dense_M            brute-force matrix of M (tiny lattices only)           PAPER.md:43-47, Eq. (2.1)
  gamma5_mul, cgnr   CG on M^dag M with M^dag = Gamma_5 M Gamma_5           PAPER.md:164 (future work there) ; pin P9

Pins (tests/test_oracle_*.py, all -m "not gpu"): direct == W form (P1); free-field closed
form and plane-wave eigen-relation (P2); gauge covariance (P3); gamma5-hermiticity and
Eqs. (2.3)/(2.10) (P4); hand-coded Wilson / Wilson-clover special cases (P5); zero-block
structure (P6); dense LU vs BiCGStab (P7); staple content of the c5 hop term (Eq. 2.8's 1/4);
mixed-precision defect correction vs dense LU (P8); CG on the normal equations and Gamma_5 M Gamma_5 = M^dag (P9);
cubic-group covariance: 90-degree rotations about the three spatial axes with the matching spinor rotation, and spatial
parity with gamma_4 (P10: pins the assignment of sigma_i to direction i, the orientation of every B_i and E_i component
against the links, and the diagonal / off-diagonal placement of the axial and vector terms).
Parity unpinned (conventions with no printed value to check, shared as input spec):
trace subtraction in F (none), the choice of Pauli basis as a whole (any basis related by a spin rotation gives an
equivalent operator), the coefficient values, the overall sign convention E_i = F_4i (a sign of c_E).

Conventions (DESIGN.md R-GAMMA): sigma_k standard Pauli; gamma_i = [[0,s_i],[s_i,0]],
gamma_4 = diag(1,1,-1,-1); a 12x12 W is W[3*alpha+a, 3*beta+b]; the paper's 2x2 block
notation is over (upper spin alpha=0,1 | lower spin alpha=2,3); a 6x6 block "sigma C" is
kron(sigma, C).  Directions mu = 0,1,2 spatial (paper's i=1,2,3), mu = 3 temporal (paper's 4).
"""
from __future__ import annotations

import numpy as np

I2 = np.eye(2, dtype=np.complex128)
SIGMA = [np.array([[0, 1], [1, 0]], dtype=np.complex128),
         np.array([[0, -1j], [1j, 0]], dtype=np.complex128),
         np.array([[1, 0], [0, -1]], dtype=np.complex128)]
Z2 = np.zeros((2, 2), dtype=np.complex128)
GAMMA = [np.block([[Z2, s], [s, Z2]]) for s in SIGMA] + [np.diag([1, 1, -1, -1]).astype(np.complex128)]
GAMMA5 = GAMMA[0] @ GAMMA[1] @ GAMMA[2] @ GAMMA[3]
EPS = np.zeros((3, 3, 3))
for _a, _b, _c in [(0, 1, 2), (1, 2, 0), (2, 0, 1)]:
    EPS[_a, _b, _c] = 1.0
    EPS[_b, _a, _c] = -1.0

# Stencil offsets of Eq. (2.2), in the term order of include/ok.h:
# 0 | +-x +-y +-z +-t | +-2x +-2y +-2z | for (i<j) in (xy),(xz),(yz): +i+j, -i-j, +i-j, -i+j
PAIRS = [(0, 1), (0, 2), (1, 2)]


def _unit(mu, s=1):
    v = [0, 0, 0, 0]
    v[mu] = s
    return np.array(v)


OFFSETS = [np.zeros(4, dtype=int)]
for _mu in range(4):
    OFFSETS += [_unit(_mu, 1), _unit(_mu, -1)]
for _i in range(3):
    OFFSETS += [_unit(_i, 2), _unit(_i, -2)]
for _i, _j in PAIRS:
    OFFSETS += [_unit(_i) + _unit(_j), -_unit(_i) - _unit(_j), _unit(_i) - _unit(_j), -_unit(_i) + _unit(_j)]
OFFSETS = np.array(OFFSETS)
assert OFFSETS.shape == (27, 4)        # 27 terms x 16 colour blocks = 432


def dag(A):
    """Hermitian conjugate of the trailing matrix ("applied in both spin and color spaces")."""
    return np.conj(np.swapaxes(A, -1, -2))


def kron(s, C):
    """6x6 block  s (x) C  for a 2x2 spin matrix s and colour matrices C[n,3,3]."""
    n = C.shape[0]
    return np.einsum("ab,nij->naibj", s, C).reshape(n, 6, 6)


def blocks(A, B, C, D):
    """12x12 matrices [[A,B],[C,D]] over (upper | lower) spin; each block [n,6,6]."""
    return np.concatenate([np.concatenate([A, B], axis=2), np.concatenate([C, D], axis=2)], axis=1)


class Oracle:
    """All fields of one gauge configuration + parameter set.

    U: links [V,4,3,3] (canonical layout, periodic, BEFORE the boundary fold)
    p: dict with dims, bc, kappa, u0, zeta, rs, cB, cE, cEE, c1..c5
    """

    def __init__(self, U, p):
        self.p = dict(p)
        self.dims = np.array(p["dims"], dtype=int)
        self.V = int(np.prod(self.dims))
        assert U.shape == (self.V, 4, 3, 3)
        n = np.arange(self.V)
        Lx, Ly, Lz, T = self.dims
        self.coords = np.stack([n % Lx, (n // Lx) % Ly, (n // (Lx * Ly)) % Lz, n // (Lx * Ly * Lz)], axis=1)
        self.U = self.fold_bc(np.asarray(U, dtype=np.complex128))

    # ------------------------------------------------------------------ geometry
    def sh(self, idx, off):
        """site indices of x + off for the sites x in idx (periodic wrap; t_{+-mu} of Eq. 2.5)."""
        c = (self.coords[idx] + np.asarray(off)[None, :]) % self.dims[None, :]
        Lx, Ly, Lz, T = self.dims
        return c[:, 0] + Lx * (c[:, 1] + Ly * (c[:, 2] + Lz * c[:, 3]))

    def fold_bc(self, U):
        """R-BC: multiply U_mu(x) by bc[mu] on the last slice of every antiperiodic axis, before
        everything else.  Fermion hops across the boundary pick up exactly one sign; closed
        loops (clover leaves) contain the boundary link with its inverse and are unchanged."""
        U = U.copy()
        for mu in range(4):
            if self.p["bc"][mu] == -1:
                last = self.coords[:, mu] == self.dims[mu] - 1
                U[last, mu] *= -1.0
        return U

    def link(self, mu, idx):
        return self.U[idx, mu]

    # ------------------------------------------------------------------ field strength
    def F(self, mu, nu, idx):
        """R-F: F_mu,nu(x) = (Q - Q^dag)/8, Q = sum of the four plaquette leaves in the mu-nu plane
        that start and end at x (counter-clockwise); anti-Hermitian, no trace subtraction."""
        U = self.link
        m, n_ = _unit(mu), _unit(nu)
        x = idx
        xpm, xpn = self.sh(x, m), self.sh(x, n_)
        xmm, xmn = self.sh(x, -m), self.sh(x, -n_)
        xmmpn, xmmmn, xpmmn = self.sh(x, -m + n_), self.sh(x, -m - n_), self.sh(x, m - n_)
        Q = U(mu, x) @ U(nu, xpm) @ dag(U(mu, xpn)) @ dag(U(nu, x))
        Q = Q + U(nu, x) @ dag(U(mu, xmmpn)) @ dag(U(nu, xmm)) @ U(mu, xmm)
        Q = Q + dag(U(mu, xmm)) @ dag(U(nu, xmmmn)) @ U(mu, xmmmn) @ U(nu, xmn)
        Q = Q + dag(U(nu, xmn)) @ U(mu, xmn) @ U(nu, xpmmn) @ dag(U(mu, x))
        return (Q - dag(Q)) / 8.0

    def B(self, i, idx):
        """B_i = (1/2) eps_ijk F_jk : B_1 = F_23, B_2 = F_31, B_3 = F_12."""
        j, k = (i + 1) % 3, (i + 2) % 3
        return self.F(j, k, idx)

    def E(self, i, idx):
        """E_i = F_4i."""
        return self.F(3, i, idx)

    def Ebar_S(self, idx):
        """Eq. (2.7):  Ebar^S_x = sum_i sigma_i E_{i,x}."""
        return sum(kron(SIGMA[i], self.E(i, idx)) for i in range(3))

    def Bbar_D(self, idx):
        """Eq. (2.7):  Bbar^D_x = i sum_i sigma_i B_{i,x}."""
        return 1j * sum(kron(SIGMA[i], self.B(i, idx)) for i in range(3))

    # ------------------------------------------------------------------ positive matrices
    def W0(self, idx):
        """Eq. (2.6)."""
        p = self.p
        n = len(idx)
        D0 = -(p["cB"] * p["zeta"] + 16 * p["c5"]) / (2 * p["u0"] ** 3) * self.Bbar_D(idx)
        S0 = -(p["cE"] * p["zeta"]) / (2 * p["u0"] ** 3) * self.Ebar_S(idx)
        mass = p["u0"] / (2 * p["kappa"]) * np.broadcast_to(np.eye(12, dtype=np.complex128), (n, 12, 12))
        return mass + blocks(D0, S0, -S0, D0)

    def S4_plus(self, idx):
        """Eq. (2.7): S^+_{4,x} = c_EE/(2 u0^4) (U_{4,x} Ebar^S_{x+4} - Ebar^S_x U_{4,x})."""
        p = self.p
        IU = kron(I2, self.link(3, idx))
        return p["cEE"] / (2 * p["u0"] ** 4) * (IU @ self.Ebar_S(self.sh(idx, _unit(3))) - self.Ebar_S(idx) @ IU)

    def W4_plus(self, idx):
        """Eq. (2.7): W^+_{4,x} = [[0, S],[S, -U_{4,x}]]."""
        S = self.S4_plus(idx)
        Z = np.zeros_like(S)
        return blocks(Z, S, S, -kron(I2, self.link(3, idx)))

    def DS_plus(self, i, idx):
        """Eq. (2.8): (D^+_{i,x}, S^+_{i,x})."""
        p = self.p
        u0 = p["u0"]
        x = idx
        xpi = self.sh(x, _unit(i))
        Ui = self.link(i, x)
        IU = kron(I2, Ui)
        sI = np.kron(SIGMA[i], np.eye(3))[None]          # sigma_i (x) 1_colour
        IB_x = kron(I2, self.B(i, x))                    # un-barred B_{i,x} = 1_2 (x) B_i
        IB_xpi = kron(I2, self.B(i, xpi))
        Bx, Bxpi = self.Bbar_D(x), self.Bbar_D(xpi)
        S = 0.5 * (p["zeta"] - 2 * p["c1"] - 12 * p["c2"]) * kron(SIGMA[i], Ui) \
            + p["c3"] / (2 * u0 ** 4) * (IU @ sI @ Bxpi - sI @ Bx @ IU + 2j * IB_x @ IU)
        D = -0.5 * (p["rs"] * p["zeta"] + 8 * p["c4"]) * IU
        st = np.zeros_like(IU)
        for j in range(3):
            for k in range(3):
                if EPS[i, j, k] != 0.0:
                    st = st + EPS[i, j, k] * kron(SIGMA[j], self.staple_up(i, k, x) - self.staple_down(i, k, x))
        D = D + 1j * p["c5"] / 4 * (u0 ** -2 - u0 ** -4) * st
        D = D + p["c5"] / u0 ** 4 * (IU @ Bxpi + Bx @ IU - 1j * sI @ (IU @ IB_xpi + IB_x @ IU))
        return D, S

    def staple_up(self, i, k, idx):
        """U_{k,x} U_{i,x+k} U^dag_{k,x+i}  (Eq. 2.8)."""
        return self.link(k, idx) @ self.link(i, self.sh(idx, _unit(k))) @ dag(self.link(k, self.sh(idx, _unit(i))))

    def staple_down(self, i, k, idx):
        """U^dag_{k,x-k} U_{i,x-k} U_{k,x-k+i}  (Eq. 2.8)."""
        xmk = self.sh(idx, -_unit(k))
        return dag(self.link(k, xmk)) @ self.link(i, xmk) @ self.link(k, self.sh(idx, -_unit(k) + _unit(i)))

    def DS_pp_ii(self, i, idx):
        """Eq. (2.9)."""
        p = self.p
        P = self.link(i, idx) @ self.link(i, self.sh(idx, _unit(i)))
        return p["c4"] / p["u0"] * kron(I2, P), (p["c1"] + 2 * p["c2"]) / (2 * p["u0"]) * kron(SIGMA[i], P)

    def S_pp_ij(self, i, j, idx):
        """Eq. (2.11)."""
        p = self.p
        P = self.link(i, idx) @ self.link(j, self.sh(idx, _unit(i))) \
            + self.link(j, idx) @ self.link(i, self.sh(idx, _unit(j)))
        return p["c2"] / (2 * p["u0"]) * kron(SIGMA[i] + SIGMA[j], P)

    def S_pm_ij(self, i, j, idx):
        """Eq. (2.12): hop to x + i - j."""
        p = self.p
        xmj = self.sh(idx, -_unit(j))
        P = self.link(i, idx) @ dag(self.link(j, self.sh(idx, -_unit(j) + _unit(i)))) \
            + dag(self.link(j, xmj)) @ self.link(i, xmj)
        return p["c2"] / (2 * p["u0"]) * kron(SIGMA[i] - SIGMA[j], P)

    # ------------------------------------------------------------------ all 27 matrices
    def precalc_W(self, idx=None):
        """W[n, 27, 12, 12] at the sites idx (default: all), term order = OFFSETS.
        Positive matrices as printed (Eqs. 2.6-2.9, 2.11, 2.12); negative ones from the
        conjugation relations (2.10) and (2.3), reading R-DAGGER ("dagger dagger" = "+ dagger")."""
        if idx is None:
            idx = np.arange(self.V)
        idx = np.asarray(idx)
        W = np.zeros((len(idx), 27, 12, 12), dtype=np.complex128)
        W[:, 0] = self.W0(idx)
        for i in range(3):
            D, S = self.DS_plus(i, idx)
            W[:, 1 + 2 * i] = blocks(D, S, S, D)
            Dm, Sm = self.DS_plus(i, self.sh(idx, -_unit(i)))                     # at x - i   (2.10)
            W[:, 2 + 2 * i] = blocks(dag(Dm), -dag(Sm), -dag(Sm), dag(Dm))
            D2, S2 = self.DS_pp_ii(i, idx)
            W[:, 9 + 2 * i] = blocks(D2, S2, S2, D2)
            D2m, S2m = self.DS_pp_ii(i, self.sh(idx, -2 * _unit(i)))              # at x - 2i  (2.10)
            W[:, 10 + 2 * i] = blocks(dag(D2m), -dag(S2m), -dag(S2m), dag(D2m))
        W[:, 7] = self.W4_plus(idx)
        xm4 = self.sh(idx, -_unit(3))
        S4m = self.S4_plus(xm4)                                                   # at x - 4   (2.10)
        Z = np.zeros_like(S4m)
        W[:, 8] = blocks(-kron(I2, dag(self.link(3, xm4))), -dag(S4m), -dag(S4m), Z)
        for q, (i, j) in enumerate(PAIRS):
            Z = np.zeros((len(idx), 6, 6), dtype=np.complex128)
            S = self.S_pp_ij(i, j, idx)
            W[:, 15 + 4 * q] = blocks(Z, S, S, Z)                                 # W^{++}_{ij,x}
            Sm = self.S_pp_ij(i, j, self.sh(idx, -_unit(i) - _unit(j)))
            W[:, 16 + 4 * q] = -dag(blocks(Z, Sm, Sm, Z))                         # W^{--}_{ij,x}   (2.3)
            S = self.S_pm_ij(i, j, idx)
            W[:, 17 + 4 * q] = blocks(Z, S, S, Z)                                 # W^{+-}_{ij,x}
            Sm = self.S_pm_ij(i, j, self.sh(idx, -_unit(i) + _unit(j)))
            W[:, 18 + 4 * q] = -dag(blocks(Z, Sm, Sm, Z))                         # W^{+-}_{ji,x}   (2.3)
        return W

    # ------------------------------------------------------------------ apply, W form
    def apply_W(self, psi, idx=None, W=None, chunk=4096):
        """Eq. (2.2): out_x = sum_o W_o(x) psi(x + o) at the sites idx.
        psi: [V,12] (or [V,12,nrhs]); W: optional precomputed [len(idx),27,12,12]."""
        if idx is None:
            idx = np.arange(self.V)
        idx = np.asarray(idx)
        out = np.zeros((len(idx),) + psi.shape[1:], dtype=np.complex128)
        for a in range(0, len(idx), chunk):
            s = idx[a:a + chunk]
            Wc = self.precalc_W(s) if W is None else W[a:a + chunk]
            for o in range(27):
                nb = psi[self.sh(s, OFFSETS[o])]
                if psi.ndim == 2:
                    out[a:a + chunk] += np.einsum("nij,nj->ni", Wc[:, o], nb)
                else:
                    out[a:a + chunk] += Wc[:, o] @ nb
        return out

    # ------------------------------------------------------------------ apply, direct form
    def apply_direct(self, psi):
        """R-DIRECT: the operator as raw gauge-link products (the paper's "Naive" inverter applies
        the action this way each iteration).  Built from covariant shifts
          (T_mu f)(x) = U_mu(x) f(x+mu),  (T_-mu f)(x) = U_mu(x-mu)^dag f(x-mu),
          D_mu = (T_mu - T_-mu)/2,  Delta_mu = T_mu + T_-mu - 2.
        Tadpole rule: every T carries 1/u0, every F carries 1/u0^4, the whole operator is
        multiplied by u0; products in which links cancel are counted after cancellation
        (two corrections below, DESIGN.md R-U0)."""
        p = self.p
        u0 = p["u0"]
        V = self.V
        allx = np.arange(V)
        psi = psi.reshape(V, 4, 3)

        def spin(G, f):                  # 4x4 spin matrix on f[V,4,3]
            return np.einsum("st,ntc->nsc", G, f)

        def col(C, f):                   # colour matrix field C[V,3,3] on f
            return np.einsum("nab,nsb->nsa", C, f)

        def Tp(mu, f):
            return col(self.link(mu, allx), f[self.sh(allx, _unit(mu))]) / u0

        def Tm(mu, f):
            xm = self.sh(allx, -_unit(mu))
            return col(dag(self.link(mu, xm)), f[xm]) / u0

        def Dc(mu, f):
            return 0.5 * (Tp(mu, f) - Tm(mu, f))

        def Lap(mu, f):
            return Tp(mu, f) + Tm(mu, f) - 2.0 * f

        Bf = [self.B(i, allx) / u0 ** 4 for i in range(3)]
        Ef = [self.E(i, allx) / u0 ** 4 for i in range(3)]
        Sig = [np.kron(I2, SIGMA[i]) for i in range(3)]            # Sigma_i = diag(s_i, s_i)
        Alp = [GAMMA[3] @ GAMMA[i] for i in range(3)]              # alpha_i = gamma_4 gamma_i

        def gD(f):                        # gamma . D
            return sum(spin(GAMMA[i], Dc(i, f)) for i in range(3))

        def Lap3(f):
            return sum(Lap(i, f) for i in range(3))

        def iSB(f):                       # i Sigma . B
            return 1j * sum(spin(Sig[i], col(Bf[i], f)) for i in range(3))

        def aE(f):                        # alpha . E
            return sum(spin(Alp[i], col(Ef[i], f)) for i in range(3))

        def g4D4(f):
            return spin(GAMMA[3], Dc(3, f))

        m0 = 1.0 / (2 * p["kappa"]) - (1.0 + 3 * p["rs"] * p["zeta"] + 18 * p["c4"])
        out = m0 * psi + g4D4(psi) - 0.5 * Lap(3, psi)
        out = out + p["zeta"] * gD(psi) - 0.5 * p["rs"] * p["zeta"] * Lap3(psi)
        out = out - 0.5 * p["cB"] * p["zeta"] * iSB(psi) - 0.5 * p["cE"] * p["zeta"] * aE(psi)
        out = out + p["c1"] * sum(spin(GAMMA[i], Dc(i, Lap(i, psi))) for i in range(3))
        out = out + p["c2"] * (gD(Lap3(psi)) + Lap3(gD(psi)))
        out = out + p["c3"] * (gD(iSB(psi)) + iSB(gD(psi)))
        out = out + p["cEE"] * (g4D4(aE(psi)) + aE(g4D4(psi)))
        out = out + p["c4"] * sum(Lap(i, Lap(i, psi)) for i in range(3))
        for i in range(3):
            for j in range(3):
                if j != i:
                    iSBi = lambda f, i=i: 1j * spin(Sig[i], col(Bf[i], f))
                    out = out + p["c5"] * (iSBi(Lap(j, psi)) + Lap(j, iSBi(psi)))
        out = u0 * out
        # R-U0 (i): T_i T_-i = 1 inside Delta_i^2 is link-free, so it carries no u0.
        out = out + u0 * p["c4"] * 3 * (2.0 - 2.0 / u0 ** 2) * psi
        # R-U0 (ii): the 3-link staples hidden in c5 {i Sigma_j B_j, Delta_i} carry u0^-2, not
        # u0^-4 -- Eq. (2.8)'s explicit (u0^-2 - u0^-4) term.
        cst = 1j * p["c5"] / 4 * (u0 ** -2 - u0 ** -4)
        for i in range(3):
            xp, xm = self.sh(allx, _unit(i)), self.sh(allx, -_unit(i))
            for j in range(3):
                for k in range(3):
                    if EPS[i, j, k] != 0.0:
                        G = self.staple_up(i, k, allx) - self.staple_down(i, k, allx)
                        out = out + cst * EPS[i, j, k] * (spin(Sig[j], col(G, psi[xp]))
                                                         - spin(Sig[j], col(dag(G[xm]), psi[xm])))
        return out.reshape(V, 12)

    # ------------------------------------------------------------------ dense M (tiny lattices)
    def dense_M(self):
        """Brute force: column c of M = apply_W(e_c).  (12V)x(12V), Eq. (2.1)."""
        n = 12 * self.V
        W = self.precalc_W()
        M = np.zeros((n, n), dtype=np.complex128)
        for c in range(n):
            e = np.zeros(n, dtype=np.complex128)
            e[c] = 1.0
            M[:, c] = self.apply_W(e.reshape(self.V, 12), W=W).reshape(n)
        return M


# ---------------------------------------------------------------------- solver
def bicgstab(apply, b, tol, maxit):
    """R-SOLVER: unpreconditioned complex BiCGStab (van der Vorst), x0 = 0, rhat = b,
    <a,b> = sum conj(a) b, stopping on ||r|| <= tol ||b|| followed by a true-residual
    check (restart from the true residual if it fails).  PAPER.md:114 names the algorithm
    ("bi-stabilized CG") and gives no listing.

    Returns (x, iters, true_relative_residual, status); status 0 ok, -3 breakdown, -4 maxit.
    """
    # reductions and scalars in fp64 whatever the storage precision of the vectors (R-SOLVER); vectors keep b's dtype
    dot = lambda a, c: complex(np.vdot(a.astype(np.complex128, copy=False), c.astype(np.complex128, copy=False)))
    bnorm = np.sqrt(dot(b, b).real)
    x = np.zeros_like(b)
    if bnorm == 0.0:
        return x, 0, 0.0, 0
    r = b.copy()
    rhat = b.copy()
    p = r.copy()
    rho = dot(rhat, r)
    status = -4
    it = 0
    bad = lambda z: (not np.isfinite(abs(z))) or abs(z) < 1e-300
    while it < maxit:
        it += 1
        v = apply(p)
        rv = dot(rhat, v)
        if bad(rv) or bad(rho):
            status = -3
            break
        alpha = rho / rv
        s = r - alpha * v
        t = apply(s)
        tt = dot(t, t).real
        if bad(tt):
            status = -3
            break
        omega = dot(t, s) / tt
        x = x + alpha * p + omega * s
        r = s - omega * t
        if np.sqrt(dot(r, r).real) <= tol * bnorm:
            rtrue = b - apply(x)
            if np.sqrt(dot(rtrue, rtrue).real) <= tol * bnorm:
                status = 0
                break
            r = rtrue
            rhat = r.copy()
            p = r.copy()
            rho = dot(rhat, r)
            continue
        if bad(omega):
            status = -3
            break
        rho_new = dot(rhat, r)
        beta = (rho_new / rho) * (alpha / omega)
        rho = rho_new
        p = r + beta * (p - omega * v)
    rtrue = b - apply(x)
    return x, it, float(np.sqrt(dot(rtrue, rtrue).real) / bnorm), status


def bicgstab_mixed(apply_hi, apply_lo, b, tol, inner_tol, maxit, max_outer=50, lo_dtype=np.complex64):
    """R-MIXED.  PAPER.md:114 only says that a mixed precision inversion is done "by calling the QOPQDP inverter or
    Dirac operation module in single or double precision, as appropriate".  Reading: classical defect correction
    (iterative refinement) around the low-precision inverter,

        x = 0 ; r = b                                   (high precision)
        repeat:  stop when ||r|| <= tol ||b||
                 e  = bicgstab(M_lo, r / ||r|| rounded to low precision, inner_tol)    (the inverter, low precision)
                 x += ||r|| e ;  r = b - M_hi x                                        (the Dirac module, high precision)

    apply_hi / apply_lo: the operator in the two precisions.  `maxit` bounds the TOTAL number of inner iterations.
    Returns (x, inner_iters_total, outer_iters, true_relative_residual, status)."""
    nrm = lambda a: float(np.sqrt(np.vdot(a, a).real))
    bnorm = nrm(b)
    x = np.zeros_like(b)
    if bnorm == 0.0:
        return x, 0, 0, 0.0, 0
    r = b.copy()
    total, outer, status = 0, 0, -4
    while True:
        rn = nrm(r)
        if rn <= tol * bnorm:
            status = 0
            break
        if outer >= max_outer or total >= maxit:
            break
        e, it, _, st = bicgstab(apply_lo, (r / rn).astype(lo_dtype), inner_tol, maxit - total)
        total += it
        outer += 1
        if st == -3:
            status = -3
            break
        x = x + rn * e.astype(b.dtype)
        r = b - apply_hi(x)
    return x, total, outer, nrm(b - apply_hi(x)) / bnorm, status


def gamma5_mul(v):
    """(Gamma_5 v)(x) = gamma_5 v(x) on a spinor field [V, 12] (gamma_5 = gamma_1 gamma_2 gamma_3 gamma_4 x 1_colour)."""
    return np.einsum("ab,nbc->nac", GAMMA5, v.reshape(-1, 4, 3)).reshape(v.shape)


def cgnr(apply, b, tol, maxit):
    """Conjugate gradient on the normal equations M^dag M x = M^dag b ("M^dag M preconditioning", named as future
    work there), with M^dag = Gamma_5 M Gamma_5 (gamma_5-hermiticity of the OK action, pin P4).
    Textbook CGNR, x0 = 0:  r = b; z = M^dag r; p = z;  loop: w = M p; alpha = <z,z>/<w,w>; x += alpha p; r -= alpha w;
    stop when ||r|| <= tol ||b|| (then true-residual check, restart from it if it fails); z' = M^dag r; beta = <z',z'>/<z,z>; p = z' + beta p.
    Returns (x, iters, true_relative_residual, status); status 0 ok, -3 breakdown, -4 maxit."""
    dag = lambda v: gamma5_mul(apply(gamma5_mul(v)))
    n2 = lambda a: float(np.vdot(a, a).real)
    bn2 = n2(b)
    x = np.zeros_like(b)
    if bn2 == 0.0:
        return x, 0, 0.0, 0
    r = b.copy()
    z = dag(r)
    p = z.copy()
    zz = n2(z)
    it, status = 0, -4
    while it < maxit:
        it += 1
        w = apply(p)
        ww = n2(w)
        if not np.isfinite(ww) or ww < 1e-300 or zz < 1e-300:
            status = -3
            break
        alpha = zz / ww
        x = x + alpha * p
        r = r - alpha * w
        if n2(r) <= tol * tol * bn2:
            rt = b - apply(x)
            if n2(rt) <= tol * tol * bn2:
                status = 0
                break
            r = rt
            z = dag(r)
            p = z.copy()
            zz = n2(z)
            continue
        z = dag(r)
        zz_new = n2(z)
        p = z + (zz_new / zz) * p
        zz = zz_new
    rt = b - apply(x)
    return x, it, float(np.sqrt(n2(rt) / bn2)), status
