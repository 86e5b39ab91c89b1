"""The pinned oracle is frozen: its outputs on a seeded 4x3x3x2 case must not drift
(values written by tests/golden/make_golden.py, which calls only oracle/)."""
import json
import os

import numpy as np

from oracle.ok_oracle import Oracle, bicgstab
from paper_1311_5029_b200 import inputs as I


def test_oracle_regression():
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "oracle_regression.json")))
    dims = tuple(g["dims"])
    U = I.near_identity_links(dims, 0.3, 1)
    plaq = I.mean_plaquette(dims, U)
    assert abs(plaq - g["plaquette"]) < 1e-14
    o = Oracle(U, I.make_params(dims, 0.10, I.tadpole_u0(plaq)))
    psi = I.gaussian_spinor(dims, 2)
    out = o.apply_W(psi)
    want = np.array([complex(*z) for z in g["out_site0"]])
    assert np.abs(out[0] - want).max() < 1e-12
    assert abs(np.linalg.norm(out) - g["out_norm"]) < 1e-10
    W = o.precalc_W(np.array([0, 17]))
    want = np.array([complex(*z) for z in g["W_site17_term1_row0"]])
    assert np.abs(W[1, 1, 0] - want).max() < 1e-14
    assert abs(np.linalg.norm(W[0]) - g["W_frobenius_site0"]) < 1e-12
    x, it, res, st = bicgstab(lambda v: o.apply_W(v), psi, 1e-10, 500)
    assert st == 0 and abs(it - g["bicgstab_iters"]) <= 1
    assert abs(np.linalg.norm(x) - g["bicgstab_x_norm"]) < 1e-8
