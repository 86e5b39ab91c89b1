"""Host-side layout logic of the reduced W storage formats (csrc/ok_sparse.cuh through ok_W_unit_index; no GPU needed),
checked against the ORACLE's precalculation matrices: the set of elements a format keeps must be exactly the structurally
non-zero ones (432 colour blocks per site, 172 vanish), every kept element must have its own slot, and the
implied copies must reproduce the oracle's W (UL = LR = D, LL = +-S; Eqs. 2.3, 2.10 for the opposite directions)."""
import numpy as np
import pytest

from oracle import ok_oracle as oo
from oracle.ok_oracle import Oracle
from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import inputs as I

UNITS = {B.OK_W_BLOCK: 260 * 9, B.OK_W_DS: 132 * 9, B.OK_W_CONJ: 70 * 9}


@pytest.fixture(scope="module")
def oracle_W():
    dims = (4, 3, 3, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    o = Oracle(U, I.make_params(dims, 0.10, 0.93))
    return o, o.precalc_W()


@pytest.mark.parametrize("fmt", [B.OK_W_BLOCK, B.OK_W_DS, B.OK_W_CONJ])
def test_layout_is_a_bijection_onto_the_nonzero_pattern(oracle_W, fmt):
    o, W = oracle_W
    pattern = np.abs(W).max(axis=0) > 0                      # [27, 12, 12]
    assert int(pattern.reshape(27, 4, 3, 4, 3).any(axis=(2, 4)).sum()) == 260
    slots = {}
    for t in range(27):
        for r in range(12):
            for c in range(12):
                u, stored, sign, conj, shift = B.ok_W_unit_index(fmt, t, r, c)
                assert (u >= 0) == bool(pattern[t, r, c]), (t, r, c)
                if u >= 0 and stored:
                    assert u not in slots, (t, r, c, slots.get(u))
                    slots[u] = (t, r, c)
    assert sorted(slots) == list(range(UNITS[fmt]))          # every unit of the record is used exactly once
    assert B.ok_W_unit_index(fmt, 27, 0, 0)[0] == -2 and B.ok_W_unit_index(0, 0, 0, 0)[0] == -2


@pytest.mark.parametrize("fmt", [B.OK_W_BLOCK, B.OK_W_DS, B.OK_W_CONJ])
def test_layout_reconstructs_the_oracle_W(oracle_W, fmt):
    """Emulate pack + unpack on the host with the index function alone and compare with the oracle's matrices."""
    o, W = oracle_W
    V = o.V
    rec = np.zeros((V, UNITS[fmt]), dtype=np.complex128)
    refs = {}
    for t in range(27):
        for r in range(12):
            for c in range(12):
                refs[t, r, c] = B.ok_W_unit_index(fmt, t, r, c)
                u, stored = refs[t, r, c][:2]
                if u >= 0 and stored:
                    rec[:, u] = W[:, t, r, c]
    back = np.zeros_like(W)
    sites = np.arange(V)
    for (t, r, c), (u, stored, sign, conj, shift) in refs.items():
        if u < 0:
            continue
        src = sites if shift < 0 else o.sh(sites, oo.OFFSETS[shift])
        v = rec[src, u]
        back[:, t, r, c] = sign * (np.conj(v) if conj else v)
    assert np.array_equal(back, W)


def test_slab_and_pauli_sizes_are_pure_host_arithmetic():
    """ok_slab_* sizes (t-slab decomposition, include/ok.h) and the OK_W_PAULI footprint need no device."""
    from paper_1311_5029_b200 import inputs as I
    dims = (20, 20, 20, 64)
    pd = I.make_params(dims, 0.10, 0.95)
    for prec, rb in ((B.OK_FP32, 4), (B.OK_FP64, 8)):
        p = B.make_params(pd, prec)
        sp = B.make_slab_params(p, 16)
        assert sp.reserved_ == B.OK_SLAB and list(sp.dims) == [20, 20, 20, 16]
        slice_bytes = 20 * 20 * 20 * 12 * 2 * rb
        assert B.ok_slab_slice_bytes(sp) == slice_bytes                      # 768 000 B at 20^3 fp32: one halo message
        assert B.ok_slab_vec_bytes(sp) == 18 * slice_bytes
        assert B.ok_W_bytes(sp) == 1024 + 20 * 20 * 20 * 16 * 27 * 144 * 2 * rb
        assert B.ok_slab_work_bytes(sp, 4, 2) > 4 * 6 * 18 * slice_bytes
        # not a slab (reserved_ = 0), or a time slice that is not a whole number of 32-site blocks: refused
        assert B.ok_slab_vec_bytes(p) == 0
        assert B.ok_slab_vec_bytes(B.make_slab_params(B.make_params(I.make_params((3, 3, 3, 8), 0.1, 0.95), prec), 4)) == 0
        q = B.make_params(pd, prec, storage=B.OK_W_PAULI)
        assert B.ok_W_bytes(q) == 1024 + 20 * 20 * 20 * 64 * 37 * 9 * 2 * rb   # 2 664 B per site in fp32 ("50 color blocks")
    assert B.ok_W_unit_index(B.OK_W_PAULI, 0, 0, 0)[0] == -2          # no element-wise layout query for this format (ok.h)
