"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (configs[2], configs[3]):
20^3 x 64, fp32, the same seeded links (eps = 0.25) and sources as the bench workloads.

The oracle cannot apply the operator to 512 000 sites in seconds, so the CUDA result is compared on SAMPLED
sites that the oracle computes one by one (Oracle.precalc_W(idx) / apply_W(psi, idx=idx), Eq. (2.2),
PAPER.md:53-55): lattice corners and faces (every wrap-around of the stencil, the antiperiodic time
boundary, the last ragged 32-site block) plus evenly spaced and pseudo-random interior sites.
BiCGStab is checked through a property that holds at any size: the residual b - M x,
evaluated by the ORACLE on the sampled sites, extrapolates to a relative residual of the order of tol.
"""
import json
import os

import numpy as np
import pytest
import torch

from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I
import okgpu as G

pytestmark = pytest.mark.gpu

DIMS = (20, 20, 20, 64)
FP32_TOL = 2e-5
NR = 12


sample_sites = I.sample_sites

# The oracle's own BiCGStab runs at these sizes (iteration count, true residual, solution on sample sites), written by
# tests/golden/make_fullsize_golden.py from oracle/ and the seeded input generators only (hours of CPU time; not rerun here).
_GDIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
GOLD = json.load(open(os.path.join(_GDIR, "fullsize_bicgstab.json")))
GOLD_X = np.load(os.path.join(_GDIR, "fullsize_x_samples.npz"))


def check_against_golden(case, dims, it, tol, xs, ncol=1):
    """north_star: "BiCGStab iteration counts must agree within +-2" (solver: PAPER.md:114) -- here against the oracle's run
    on the same seeds at the full size; and the solution on the golden's sample sites.  Two iterates that both satisfy
    || b - M x || <= tol || b || differ by at most cond(M) 2 tol relative to || x ||; cond(M) of these fields is O(10)
    (34 BiCGStab iterations to 1e-6), the measured difference is recorded by the assert message."""
    g = GOLD[case]
    assert g["dims"] == list(dims) and g["tol"] == tol and len(g["columns"]) == ncol
    its = [c["iters"] for c in g["columns"]]
    assert all(c["status"] == 0 and c["true_resid"] <= tol for c in g["columns"])
    assert abs(it - max(its)) <= 2, (it, its)                 # the library reports the slowest column
    idx = sample_sites(dims, n_even=g["sample"]["n_even"], n_rand=g["sample"]["n_rand"])
    want = GOLD_X[case]                                        # [sites, columns, 12]
    assert want.shape == (len(idx), ncol, 12)
    got = xs[idx] if ncol == 1 else np.moveaxis(xs[idx], 2, 1)
    got = got.reshape(want.shape)
    for j in range(ncol):
        d = np.linalg.norm(got[:, j] - want[:, j]) / np.linalg.norm(want[:, j])
        assert d <= 30 * tol, (case, j, d)


@pytest.fixture(scope="module")
def big():
    out = {}
    for seed in (5, 7):                                          # configs[2] and configs[3] gauge seeds
        U = I.near_identity_links(DIMS, 0.25, seed)
        pd = I.make_params(DIMS, 0.10, I.tadpole_u0(I.mean_plaquette(DIMS, U)))
        out[seed] = (U, pd, Oracle(U, pd))
    return out


def sampled_rel_l2(got, want):
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def sampled_resid_bound(tol, o, xs, b, idx, W):
    """Bound on the oracle-evaluated residual of an fp32 solution, extrapolated from the sites idx (R-RESID):
    tol (asserted on the library's own `resid`) widened by the sampling error of the extrapolation -- the residual's 12 n
    complex components are a sample of an approximately Gaussian field, so the estimate of its norm scatters by 1/sqrt(24 n)
    (3 sigma taken) -- plus the fp32-operator slack of G.fp32_operator_slack on the same sites."""
    return tol * (1.0 + 3.0 / np.sqrt(24.0 * len(idx))) + G.fp32_operator_slack(o, xs, b, idx=idx, W=W)


def test_fullsize_single_rhs_apply_and_solve(big):
    U, pd, o = big[5]
    p = B.make_params(pd, B.OK_FP32)
    idx = sample_sites(DIMS)
    W = G.precalc(p, U)
    # W on the sampled sites, element by element (fp32 rounding of the fp64 precalc)
    want_W = o.precalc_W(idx)
    canon = torch.empty((o.V, 27, 12, 12), dtype=torch.complex64, device=G.DEV)
    B.ok_unpack_W(W, canon)
    got_W = canon[torch.from_numpy(idx).to(G.DEV)].cpu().numpy().astype(np.complex128)
    del canon
    assert np.abs(got_W - want_W).max() <= 2e-7 * np.abs(want_W).max()
    # apply: Gaussian source seed 6 (the bench workload)
    psi = I.gaussian_spinor(DIMS, 6)
    got = G.apply(p, W, psi)[idx]
    want = o.apply_W(psi, idx=idx, W=want_W)
    assert sampled_rel_l2(got, want) <= FP32_TOL
    assert G.per_site_rel_err(got, want) <= 10 * FP32_TOL          # fp32: every sampled site individually close
    # solve to 1e-6; the oracle evaluates the residual on the sampled sites
    G.workspace(p)
    src = G.pack_spinor(p, psi)
    x = B.alloc_vec(p)
    tol = 1e-6
    st, it, res = B.ok_bicgstab(W, src, x, tol, 2000, raise_on_fail=False)
    assert st == 0 and res <= tol
    xs = G.unpack_spinor(p, x, psi.shape)
    check_against_golden("cfg2", DIMS, it, tol, xs)
    r = psi[idx] - o.apply_W(xs, idx=idx, W=want_W)
    est = np.sqrt(o.V / len(idx)) * np.linalg.norm(r) / np.linalg.norm(psi)
    assert est <= sampled_resid_bound(tol, o, xs, psi, idx, want_W), est


def test_fullsize_12rhs_apply_and_solve(big):
    U, pd, o = big[7]
    p = B.make_params(pd, B.OK_FP32, nrhs=NR)
    idx = sample_sites(DIMS, n_even=192, n_rand=192)
    W = G.precalc(p, U)
    want_W = o.precalc_W(idx)
    # Gaussian block: every site of the sample is exercised
    psi = np.stack([I.gaussian_spinor(DIMS, 60 + j) for j in range(NR)], axis=2)
    got = G.apply(p, W, psi)[idx]
    want = o.apply_W(psi, idx=idx, W=want_W)
    num = np.linalg.norm((got - want).reshape(-1, NR), axis=0)
    den = np.linalg.norm(want.reshape(-1, NR), axis=0)
    assert float((num / den).max()) <= FP32_TOL
    del psi, got
    # configs[3]: the 12 point sources at the origin
    b = np.stack([I.point_source(DIMS, site=0, comp=j) for j in range(NR)], axis=2)
    G.workspace(p)
    src = G.pack_spinor(p, b)
    x = B.alloc_vec(p)
    tol = 1e-6
    st, it, res = B.ok_bicgstab(W, src, x, tol, 2000, raise_on_fail=False)
    assert st == 0 and res <= tol
    xs = G.unpack_spinor(p, x, b.shape)
    check_against_golden("cfg3", DIMS, it, tol, xs, ncol=NR)
    # residual by the oracle: exactly on the origin's neighbourhood (where b lives and r is largest), and on a uniform
    # random sample of the remaining sites, extrapolated to the whole lattice
    rng = range(-3, 4)
    near = np.unique(np.concatenate([o.sh(np.array([0]), np.array(off)) for off in
                                     [(dx, dy, dz, dt) for dx in rng for dy in rng for dz in rng for dt in rng]]))
    rn = b[near] - o.apply_W(xs, idx=near)
    far = np.setdiff1d(np.random.default_rng(3).integers(0, o.V, 768), near)
    rf = b[far] - o.apply_W(xs, idx=far)
    n2 = np.linalg.norm(rn.reshape(-1, NR), axis=0) ** 2
    f2 = (o.V - len(near)) / len(far) * np.linalg.norm(rf.reshape(-1, NR), axis=0) ** 2
    est = np.sqrt(n2 + f2)                                                   # ||b_j|| = 1
    # R-RESID for the split-fp16 operands (9 units of 2^-24 |W||x| against the 2 of the fp32 path, tests/test_gpu_mrhs.py);
    # the near part is exact, the far part (a minor share of the norm) carries the sampling error
    sl_n = G.fp32_operator_slack(o, xs, b, idx=near) / np.sqrt(o.V / len(near))
    sl_f = G.fp32_operator_slack(o, xs, b, idx=far) * np.sqrt((o.V - len(near)) / o.V)
    bound = tol * (1.0 + 3.0 / np.sqrt(24.0 * len(far))) + 4.5 * np.sqrt(sl_n ** 2 + sl_f ** 2)
    assert np.all(est <= bound), (est, bound)


@pytest.mark.parametrize("fmt", [B.OK_W_DS, B.OK_W_CONJ, B.OK_W_PAULI])
def test_fullsize_reduced_formats_apply_and_mixed_solve(big, fmt):
    """The reduced W storage formats and the mixed-precision inversion (item 3) at the
    bench size: sampled-site parity of the fp32 apply, then ok_bicgstab_mixed(W64, W32) to 1e-10 with the residual
    evaluated by the oracle (fp64) on sampled sites."""
    U, pd, o = big[5]
    idx = sample_sites(DIMS)
    want_W = o.precalc_W(idx)
    p32 = B.make_params(pd, B.OK_FP32, storage=fmt)
    p64 = B.make_params(pd, B.OK_FP64, storage=fmt)
    W32 = G.precalc(p32, U)
    psi = I.gaussian_spinor(DIMS, 6)
    got = G.apply(p32, W32, psi)[idx]
    want = o.apply_W(psi, idx=idx, W=want_W)
    assert sampled_rel_l2(got, want) <= FP32_TOL
    W64 = G.precalc(p64, U)
    got64 = G.apply(p64, W64, psi)[idx]
    assert G.per_site_rel_err(got64, want) <= 1e-12
    need = B.ok_mixed_work_bytes(p64)
    ws = B.alloc_bytes(need, G.DEV)
    B.ok_set_workspace(ws, need)
    src = G.pack_spinor(p64, psi)
    x = B.alloc_vec(p64)
    tol = 1e-10
    st, it, outer, res = B.ok_bicgstab_mixed(W64, W32, src, x, tol, 1e-4, 2000, 50, raise_on_fail=False)
    assert st == 0 and res <= tol and 2 <= outer <= 6 and 20 <= it <= 400
    xs = G.unpack_spinor(p64, x, psi.shape)
    r = psi[idx] - o.apply_W(xs, idx=idx, W=want_W)
    est = np.sqrt(o.V / len(idx)) * np.linalg.norm(r) / np.linalg.norm(psi)
    assert est <= tol * (1.0 + 3.0 / np.sqrt(24.0 * len(idx))), est       # fp64 operator on both sides: sampling error only
    B.ok_set_workspace(None)


def test_fullsize_config5_haar_32x32x32x64():
    """BASELINE.json configs[4]: 32^3 x 64 (2 097 152 sites), fp32 W (65 GB), Haar-random links seed 8, kappa 0.08, u0 = 1
    (DESIGN.md R-U0HAAR): sampled-site apply parity, and the BiCGStab solution's residual evaluated by the oracle on sampled
    sites (the oracle computes W on the fly for the sites it is asked about)."""
    dims = (32, 32, 32, 64)
    U = I.haar_links(dims, 8)
    plaq = I.mean_plaquette(dims, U)
    u0 = I.tadpole_u0(plaq)
    assert abs(plaq) < 0.01 and u0 == 1.0
    pd = I.make_params(dims, 0.08, u0)
    o = Oracle(U, pd)
    p = B.make_params(pd, B.OK_FP32)
    idx = sample_sites(dims, n_even=256, n_rand=256)
    want_W = o.precalc_W(idx)
    W = G.precalc(p, U)
    psi = I.gaussian_spinor(dims, 9)
    got = G.apply(p, W, psi)[idx]
    want = o.apply_W(psi, idx=idx, W=want_W)
    assert sampled_rel_l2(got, want) <= FP32_TOL
    G.workspace(p)
    src = G.pack_spinor(p, psi)
    x = B.alloc_vec(p)
    tol = 1e-6
    st, it, res = B.ok_bicgstab(W, src, x, tol, 2000, raise_on_fail=False)
    assert st == 0 and res <= tol                             # strongly diagonally dominant at kappa = 0.08
    xs = G.unpack_spinor(p, x, psi.shape)
    check_against_golden("cfg4", dims, it, tol, xs)
    r = psi[idx] - o.apply_W(xs, idx=idx, W=want_W)
    est = np.sqrt(o.V / len(idx)) * np.linalg.norm(r) / np.linalg.norm(psi)
    assert est <= sampled_resid_bound(tol, o, xs, psi, idx, want_W), est


def test_fullsize_t_slabs_equal_the_whole_lattice(big):
    """The t-slab decomposition at BASELINE configs[2]'s size, 4 slabs of 16 time slices on one GPU: every slab's W
    (sampled blocks) and the slab apply equal the unsharded CUDA result bit for bit; ok_slab_bicgstab reproduces the oracle's
    iteration count (+-2) and solution (golden cfg2)."""
    from paper_1311_5029_b200 import slab as S
    U, pd, o = big[5]
    p = B.make_params(pd, B.OK_FP32)
    W = G.precalc(p, U)
    psi = I.gaussian_spinor(DIMS, 6)
    whole = G.apply(p, W, psi)
    B.ok_forget_W(W)
    del W
    torch.cuda.empty_cache()
    nslab = 4
    ranges = S.slab_ranges(DIMS[3], nslab)
    slab = B.make_slab_params(p, ranges[0][1])
    plocal = B.make_params(dict(pd, dims=DIMS[:3] + (ranges[0][1],)), B.OK_FP32)
    work = B.alloc_bytes(B.ok_slab_work_bytes(slab, nslab, 1), G.DEV)
    B.ok_set_stream(None)
    B.ok_set_workspace(work, work.numel())
    Ws, src = [], []
    for t0, Tl in ranges:
        Wt = B.alloc_W(slab, G.DEV)
        B.ok_slab_precalc_W(G.to_dev(S.link_window(U, DIMS, t0, Tl), torch.complex128), slab, DIMS[3], t0, Wt)
        Ws.append(Wt)
        v = torch.zeros(B.ok_slab_vec_bytes(slab), dtype=torch.uint8, device=G.DEV)
        B.ok_pack_spinor(plocal, G.to_dev(S.spinor_slab(psi, DIMS, t0, Tl), torch.complex64), S.interior(slab, v))
        src.append(v)
    for i in range(nslab):
        lo, first, last, hi = S.halo_views(slab, src[i])
        lo.copy_(S.halo_views(slab, src[(i - 1) % nslab])[2])
        hi.copy_(S.halo_views(slab, src[(i + 1) % nslab])[1])
    sites = DIMS[0] * DIMS[1] * DIMS[2]
    got = []
    for Wt, v in zip(Ws, src):
        out = torch.zeros_like(v)
        B.ok_slab_dirac_apply(Wt, v, out)
        canon = torch.empty((ranges[0][1] * sites, 12), dtype=torch.complex64, device=G.DEV)
        B.ok_unpack_spinor(plocal, S.interior(slab, out), canon)
        got.append(canon)
    torch.cuda.synchronize()
    got = torch.cat(got).cpu().numpy().astype(np.complex128)
    assert np.array_equal(got, whole)
    xs = [torch.zeros_like(v) for v in src]
    tol = 1e-6
    st, it, res = B.ok_slab_bicgstab(Ws, src, xs, tol, 2000, raise_on_fail=False)
    assert st == 0 and res <= tol
    xg = []
    for v in xs:
        canon = torch.empty((ranges[0][1] * sites, 12), dtype=torch.complex64, device=G.DEV)
        B.ok_unpack_spinor(plocal, S.interior(slab, v), canon)
        xg.append(canon)
    torch.cuda.synchronize()
    check_against_golden("cfg2", DIMS, it, tol, torch.cat(xg).cpu().numpy().astype(np.complex128))
    B.ok_set_workspace(None)
