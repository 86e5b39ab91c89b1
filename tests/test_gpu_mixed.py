"""Mixed-precision inversion (DESIGN.md R-MIXED) against the CPU oracle.

ok_bicgstab_mixed = defect correction around the fp32 BiCGStab with the fp64 and the fp32 precalculation matrices both
resident.  Oracle side: oracle.bicgstab_mixed with the fp64 W and its complex64 rounding (pinned against dense LU, P8).
Bars: fp64 true residual <= tol (evaluated by the oracle's fp64 operator too), the solution equals the oracle's within
10 tol, the number of corrections agrees within 1 and the total inner iteration count within 2 per correction.
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


def setup(dims, eps=0.3, seed=1, kappa=0.10):
    U = I.near_identity_links(dims, eps, seed)
    pd = I.make_params(dims, kappa, I.tadpole_u0(I.mean_plaquette(dims, U)))
    return U, pd, Oracle(U, pd)


def lo_apply(o, W32):
    idx = np.arange(o.V)
    nbr = [o.sh(idx, off) for off in oo.OFFSETS]

    def f(v):
        out = np.zeros_like(v)
        for t in range(27):
            out += np.einsum("nij,nj->ni", W32[:, t], v[nbr[t]])
        return out.astype(np.complex64)
    return f


def mixed_workspace(p):
    need = B.ok_mixed_work_bytes(p)
    buf = B.alloc_bytes(need, G.DEV)
    B.ok_set_workspace(buf, need)
    B.ok_set_stream(None)
    return buf


@pytest.mark.parametrize("storage", [(B.OK_W_DENSE, B.OK_W_DENSE), (B.OK_W_DS, B.OK_W_DS), (B.OK_W_DENSE, B.OK_W_BLOCK)])
@pytest.mark.parametrize("dims,tol,inner", [((4, 4, 4, 8), 1e-10, 1e-4), ((4, 3, 3, 2), 1e-12, 1e-3)])
def test_mixed_vs_oracle(dims, tol, inner, storage):
    U, pd, o = setup(dims)
    p64 = B.make_params(pd, B.OK_FP64, storage=storage[0])
    p32 = B.make_params(pd, B.OK_FP32, storage=storage[1])
    G.workspace(p64)
    W64 = G.precalc(p64, U)
    W32 = G.precalc(p32, U)
    b = I.gaussian_spinor(dims, 2)
    ws = mixed_workspace(p64)
    src = G.pack_spinor(p64, b)
    x = B.alloc_vec(p64)
    st, it, outer, res = B.ok_bicgstab_mixed(W64, W32, src, x, tol, inner, 2000, 50, raise_on_fail=False)
    assert st == 0 and res <= tol
    xs = G.unpack_spinor(p64, x, b.shape)
    Wc = o.precalc_W()
    hi = lambda v: o.apply_W(v, W=Wc)
    assert np.linalg.norm(b - hi(xs)) / np.linalg.norm(b) <= 1.01 * tol          # the oracle's operator agrees it is solved
    xo, ito, outo, reso, sto = oo.bicgstab_mixed(hi, lo_apply(o, Wc.astype(np.complex64)), b, tol, inner, 2000, 50)
    assert sto == 0
    assert abs(outer - outo) <= 1 and abs(it - ito) <= 2 * max(outer, outo) + 2
    assert G.rel_l2(xs, xo) <= 10 * tol
    # bit-reproducible, and the budget / argument errors
    x2 = B.alloc_vec(p64)
    again = B.ok_bicgstab_mixed(W64, W32, src, x2, tol, inner, 2000, 50, raise_on_fail=False)
    assert again == (st, it, outer, res) and torch.equal(x, x2)
    st3, it3, out3, res3 = B.ok_bicgstab_mixed(W64, W32, src, x2, tol, inner, 3, 50, raise_on_fail=False)
    assert st3 == -4 and it3 == 3 and res3 > tol
    assert B.ok_bicgstab_mixed(W32, W64, src, x2, tol, inner, 100, 50, raise_on_fail=False)[0] == -1      # precisions swapped
    del ws


def test_mixed_zero_rhs_and_workspace_check():
    dims = (4, 3, 3, 2)
    U, pd, o = setup(dims)
    p64, p32 = B.make_params(pd, B.OK_FP64), B.make_params(pd, B.OK_FP32)
    G.workspace(p64)
    W64, W32 = G.precalc(p64, U), G.precalc(p32, U)
    ws = mixed_workspace(p64)
    src = G.pack_spinor(p64, np.zeros((o.V, 12), dtype=np.complex128))
    x = B.alloc_vec(p64)
    assert B.ok_bicgstab_mixed(W64, W32, src, x, 1e-10, 1e-4, 100, 10, raise_on_fail=False) == (0, 0, 0, 0.0)
    assert np.all(G.unpack_spinor(p64, x, (o.V, 12)) == 0)
    small = B.alloc_bytes(4096, G.DEV)
    B.ok_set_workspace(small, 4096)
    assert B.ok_bicgstab_mixed(W64, W32, src, x, 1e-10, 1e-4, 100, 10, raise_on_fail=False)[0] == -5
    del ws
