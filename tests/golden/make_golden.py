"""Writes tests/golden/oracle_regression.json.  Calls ONLY oracle/ and the seeded input generators
(never the CUDA path).  The stored numbers are not pins (the pins are in tests/test_oracle_pins.py);
they freeze the pinned oracle so that a later change to its arithmetic is noticed and must be
justified in the commit message.

Run from the repo root:  python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.ok_oracle import Oracle, bicgstab  # noqa: E402
from paper_1311_5029_b200 import inputs as I  # noqa: E402


def main():
    dims = (4, 3, 3, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    plaq = I.mean_plaquette(dims, U)
    u0 = I.tadpole_u0(plaq)
    o = Oracle(U, I.make_params(dims, 0.10, u0))
    psi = I.gaussian_spinor(dims, 2)
    out = o.apply_W(psi)
    W = o.precalc_W(np.array([0, 17]))
    x, it, res, st = bicgstab(lambda v: o.apply_W(v), psi, 1e-10, 500)
    rec = {
        "_what": "oracle outputs, config-1 recipe on a 4x3x3x2 lattice (eps=0.3, link seed 1, source seed 2, kappa 0.10, OK-like v1)",
        "dims": dims, "plaquette": plaq, "u0": u0,
        "out_site0": [[z.real, z.imag] for z in out[0]],
        "out_norm": float(np.linalg.norm(out)),
        "W_site17_term1_row0": [[z.real, z.imag] for z in W[1, 1, 0]],
        "W_frobenius_site0": float(np.linalg.norm(W[0])),
        "bicgstab_iters": it, "bicgstab_x_norm": float(np.linalg.norm(x)),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    json.dump(rec, open(path, "w"), indent=1)
    print("wrote", path, "iters", it, "res", res)


if __name__ == "__main__":
    main()
