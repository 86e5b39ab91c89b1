"""Seeded synthetic inputs for the OK-action hot path.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's
tests.  It contains no arithmetic of the method (no W, no Dirac apply, no solver): only
random numbers, SU(3) link generators, sources, the mean plaquette that fixes the input
parameter u0, and random gauge transformations used as test stimuli.

Everything is numpy/fp64 on the host; the generated arrays are handed to both sides.

Conventions (canonical/external layouts):
  site index  n = x + Lx*(y + Ly*(z + Lz*t)),  dims = (Lx, Ly, Lz, T)
  links       U[n, mu, a, b]   complex128, U_mu(x) = link from x to x+mu_hat, mu=0..3 (3 = time)
  spinor      psi[n, 3*alpha + a] complex128 (alpha spin 0..3, a colour 0..2)

RNG: counter based, order independent.
  u64(seed, stream, k) = splitmix64(seed*2^40 + stream*2^32 + k)
  uniform(k)  = (u64 >> 11 + 0.5) * 2^-53                         in (0,1)
  normal(j)   = sqrt(-2 ln uniform(2j)) * cos(2 pi uniform(2j+1))  (Box-Muller, cosine branch)
  link index  j = (site*4 + mu)*8 + a        (a = Gell-Mann component 0..7; Haar: see haar_links)
  spinor index j = (site*12 + comp)*2 + {0: re, 1: im}
"""
from __future__ import annotations

import numpy as np

STREAM_LINKS = 1
STREAM_SPINOR = 2
STREAM_GAUGE_XFORM = 3

# "OK-like v1": stand-in coefficient set.  The paper's tree-level
# tadpole-improved values come from its Refs. [5],[7], which are not
# available; all twelve are caller inputs of the method, so any fixed non-degenerate set
# exercises every term.
OK_LIKE_V1 = dict(zeta=1.0, rs=1.0, cB=1.0, cE=1.0, cEE=-0.05,
                  c1=-0.15, c2=-0.03, c3=0.04, c4=0.02, c5=0.005)

WILSON = dict(zeta=1.0, rs=1.0, cB=0.0, cE=0.0, cEE=0.0,
              c1=0.0, c2=0.0, c3=0.0, c4=0.0, c5=0.0)


# --------------------------------------------------------------------------- RNG
def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output per 64-bit counter value (vectorised, wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x.astype(np.uint64) + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def _uniform(seed: int, stream: int, k: np.ndarray) -> np.ndarray:
    base = np.uint64((int(seed) << 40) + (int(stream) << 32))
    with np.errstate(over="ignore"):
        u = splitmix64(base + k.astype(np.uint64))
    return ((u >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


def normal(seed: int, stream: int, j: np.ndarray) -> np.ndarray:
    """Standard normal deviate number j of (seed, stream); j may be any integer array < 2^31."""
    j = np.asarray(j, dtype=np.uint64)
    u1 = _uniform(seed, stream, 2 * j)
    u2 = _uniform(seed, stream, 2 * j + 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# --------------------------------------------------------------------------- geometry
def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def site_coords(dims) -> np.ndarray:
    """[V,4] integer coordinates (x,y,z,t) of site n."""
    Lx, Ly, Lz, T = dims
    n = np.arange(volume(dims))
    return np.stack([n % Lx, (n // Lx) % Ly, (n // (Lx * Ly)) % Lz, n // (Lx * Ly * Lz)], axis=1)


def shifted_sites(dims, offset) -> np.ndarray:
    """Index array s with s[n] = index of site x_n + offset (periodic wrap)."""
    c = (site_coords(dims) + np.asarray(offset)[None, :]) % np.asarray(dims)[None, :]
    Lx, Ly, Lz, T = dims
    return c[:, 0] + Lx * (c[:, 1] + Ly * (c[:, 2] + Lz * c[:, 3]))


# --------------------------------------------------------------------------- SU(3)
def gell_mann() -> np.ndarray:
    lam = np.zeros((8, 3, 3), dtype=np.complex128)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1] = -1j; lam[1][1, 0] = 1j
    lam[2][0, 0] = 1; lam[2][1, 1] = -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2] = -1j; lam[4][2, 0] = 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2] = -1j; lam[6][2, 1] = 1j
    lam[7][0, 0] = lam[7][1, 1] = 1 / np.sqrt(3); lam[7][2, 2] = -2 / np.sqrt(3)
    return lam


def reunitarize(U: np.ndarray) -> np.ndarray:
    """Project [...,3,3] to SU(3): normalise row 0, Gram-Schmidt row 1, row 2 = conj(row0 x row1)."""
    r0 = U[..., 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
    r1 = U[..., 1, :]
    r1 = r1 - np.sum(np.conj(r0) * r1, axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def near_identity_links(dims, eps: float, seed: int) -> np.ndarray:
    """U = exp(i eps H), H = sum_a xi_a lambda_a / 2, xi_a ~ N(0,1); reunitarised (configs 1-4)."""
    V = volume(dims)
    j = np.arange(V * 4 * 8, dtype=np.uint64)
    xi = normal(seed, STREAM_LINKS, j).reshape(V, 4, 8)
    H = 0.5 * np.einsum("nma,aij->nmij", xi, gell_mann())
    w, vec = np.linalg.eigh(H)
    U = np.einsum("nmik,nmk,nmjk->nmij", vec, np.exp(1j * eps * w), np.conj(vec))
    return reunitarize(U)


def haar_links(dims, seed: int) -> np.ndarray:
    """Haar-random SU(3) links (config 5): QR of a complex Ginibre matrix, phases fixed by
    R's diagonal, divided by det^(1/3).  Normal index j = ((site*4+mu)*9 + 3*a + b)*2 + {re,im}."""
    V = volume(dims)
    j = np.arange(V * 4 * 9 * 2, dtype=np.uint64)
    g = normal(seed, STREAM_LINKS, j).reshape(V, 4, 3, 3, 2)
    return _haar_from_ginibre(g[..., 0] + 1j * g[..., 1])


def _haar_from_ginibre(Z: np.ndarray) -> np.ndarray:
    Q, R = np.linalg.qr(Z)
    d = np.diagonal(R, axis1=-2, axis2=-1)
    Q = Q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(Q)
    Q = Q / np.exp(1j * np.angle(det) / 3.0)[..., None, None]
    return Q


def unit_links(dims) -> np.ndarray:
    """Free field: all U = 1."""
    U = np.zeros((volume(dims), 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def random_gauge_transform(dims, seed: int) -> np.ndarray:
    """g[n] Haar SU(3) per site (pin P3 stimulus)."""
    V = volume(dims)
    j = np.arange(V * 9 * 2, dtype=np.uint64)
    g = normal(seed, STREAM_GAUGE_XFORM, j).reshape(V, 3, 3, 2)
    return _haar_from_ginibre(g[..., 0] + 1j * g[..., 1])


def gauge_transform_links(dims, U: np.ndarray, g: np.ndarray) -> np.ndarray:
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger."""
    out = np.empty_like(U)
    for mu in range(4):
        off = [0, 0, 0, 0]; off[mu] = 1
        gs = g[shifted_sites(dims, off)]
        out[:, mu] = np.einsum("nij,njk,nlk->nil", g, U[:, mu], np.conj(gs))
    return out


def gauge_transform_spinor(psi: np.ndarray, g: np.ndarray) -> np.ndarray:
    """psi'(x) = g(x) psi(x) acting on colour."""
    V = psi.shape[0]
    return np.einsum("nab,nsb->nsa", g, psi.reshape(V, 4, 3)).reshape(V, 12)


# --------------------------------------------------------------------------- sources
def gaussian_spinor(dims, seed: int) -> np.ndarray:
    V = volume(dims)
    j = np.arange(V * 12 * 2, dtype=np.uint64)
    g = normal(seed, STREAM_SPINOR, j).reshape(V, 12, 2)
    return g[..., 0] + 1j * g[..., 1]


def point_source(dims, site: int = 0, comp: int = 0) -> np.ndarray:
    psi = np.zeros((volume(dims), 12), dtype=np.complex128)
    psi[site, comp] = 1.0
    return psi


def sample_sites(dims, n_even: int = 384, n_rand: int = 384, seed: int = 11) -> np.ndarray:
    """Sorted site indices on which full-size results are compared with the oracle: the lattice corners and faces
    (every wrap-around of the stencil, the antiperiodic time boundary), the last 40 sites of the site order (the ragged
    last block), evenly spaced sites and pseudo-random interior sites.  A test stimulus only."""
    Lx, Ly, Lz, T = dims
    V = volume(dims)

    def site(x, y, z, t):
        return x + Lx * (y + Ly * (z + Lz * t))

    s = set()
    for x in (0, 1, Lx - 2, Lx - 1):
        for y in (0, 1, Ly - 2, Ly - 1):
            for z in (0, 1, Lz - 2, Lz - 1):
                for t in (0, 1, T - 2, T - 1):
                    s.add(site(x, y, z, t))
    s.update(range(V - 40, V))
    s.update((np.arange(n_even) * (V // n_even) + 7).tolist())
    s.update(np.random.default_rng(seed).integers(0, V, n_rand).tolist())
    return np.array(sorted(s), dtype=np.int64)


# --------------------------------------------------------------------------- u0
def mean_plaquette(dims, U: np.ndarray) -> float:
    """(1/6V) sum_x sum_{mu<nu} (1/3) Re Tr U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag,
    periodic links (before any boundary-condition fold)."""
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            om = [0, 0, 0, 0]; om[mu] = 1
            on = [0, 0, 0, 0]; on[nu] = 1
            A = U[:, mu]
            B = U[shifted_sites(dims, om), nu]
            C = U[shifted_sites(dims, on), mu]
            D = U[:, nu]
            tot += np.einsum("nij,njk,nlk,nil->", A, B, np.conj(C), np.conj(D)).real
    return float(tot / (6 * 3 * volume(dims)))


def tadpole_u0(plaq: float) -> float:
    """u0 = plaq^(1/4); reading S6: u0 = 1 whenever the mean plaquette <= 0.1 (Haar links)."""
    return 1.0 if plaq <= 0.1 else float(plaq ** 0.25)


def make_params(dims, kappa: float, u0: float, coeffs=None, bc=(1, 1, 1, -1)) -> dict:
    p = dict(dims=tuple(int(d) for d in dims), bc=tuple(int(b) for b in bc),
             kappa=float(kappa), u0=float(u0))
    p.update(OK_LIKE_V1 if coeffs is None else coeffs)
    return p
