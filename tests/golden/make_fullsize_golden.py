#!/usr/bin/env python
"""Writes tests/golden/fullsize_bicgstab.json (+ fullsize_x_samples.npz): the ORACLE's BiCGStab runs at BASELINE.json's
full sizes, against which tests/test_gpu_fullsize.py checks the CUDA path's iteration count (+-2, north_star), true
residual and solution.  Calls only oracle/ and the seeded input generators (paper_1311_5029_b200/inputs.py); nothing here
comes from the CUDA path.

    python tests/golden/make_fullsize_golden.py [--cases cfg2,cfg3,cfg4] [--workers N]

Cases (solver: PAPER.md:114, reading R-SOLVER; operator: Eq. (2.2)):
  cfg2  BASELINE configs[2]: 20^3 x 64, links eps = 0.25 seed 5, Gaussian source seed 6, kappa 0.10, tol 1e-6
  cfg3  BASELINE configs[3]: 20^3 x 64, links eps = 0.25 seed 7, the 12 spin-colour point sources at the origin, tol 1e-6,
        one oracle.bicgstab per column
  cfg4  BASELINE configs[4]: 32^3 x 64, Haar links seed 8, kappa 0.08, u0 = 1, Gaussian source seed 9, tol 1e-6

The oracle's arithmetic is untouched: oracle.bicgstab runs as it stands; its `apply` argument evaluates
Oracle.apply_W on contiguous site ranges in a pool of forked worker processes and concatenates the pieces (the sum over
the 27 terms of a site never crosses a range).  cfg2/cfg3 keep the fp64 W of all sites in shared memory (31.9 GB);
cfg4's W (130 GB) does not fit this host, so there the workers rebuild W for their sites at every apply
(Oracle.apply_W with W=None), which is the same arithmetic, slower.
"""
from __future__ import annotations

import argparse
import json
import mmap
import multiprocessing as mp
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import ok_oracle as oo  # noqa: E402
from paper_1311_5029_b200 import inputs as I  # noqa: E402

G = {}      # worker globals (inherited by fork)


def shared_array(shape, dtype):
    n = int(np.prod(shape)) * np.dtype(dtype).itemsize
    return np.frombuffer(mmap.mmap(-1, n), dtype=dtype).reshape(shape)


def _pre(a, b):
    o, W = G["o"], G["W"]
    for s in range(a, b, 2048):
        e = min(b, s + 2048)
        W[s:e] = o.precalc_W(np.arange(s, e))
    return b - a


def _app(a, b):
    o, W = G["o"], G["W"]
    G["out"][a:b] = o.apply_W(G["psi"], idx=np.arange(a, b), W=None if W is None else W[a:b], chunk=2048)
    return b - a


def ranges(V, n):
    step = (V + n - 1) // n
    return [(a, min(V, a + step)) for a in range(0, V, step)]


def run_case(name, dims, links, kappa, sources, tol, workers, store_W, n_even, n_rand):
    t0 = time.time()
    U = links()
    plaq = I.mean_plaquette(dims, U)
    u0 = I.tadpole_u0(plaq)
    pd = I.make_params(dims, kappa, u0)
    o = oo.Oracle(U, pd)
    V = o.V
    G.update(o=o, W=shared_array((V, 27, 12, 12), np.complex128) if store_W else None,
             psi=shared_array((V, 12), np.complex128), out=shared_array((V, 12), np.complex128))
    t_pre = None
    napply = [0]
    with mp.get_context("fork").Pool(workers) as pool:
        if store_W:
            t1 = time.time()
            pool.starmap(_pre, ranges(V, workers * 8))
            t_pre = time.time() - t1
            print(f"[{name}] oracle precalc_W of {V} sites: {t_pre:.1f} s on {workers} workers", flush=True)

        def apply(v):
            G["psi"][:] = v
            pool.starmap(_app, ranges(V, workers * 4))
            napply[0] += 1
            return G["out"].copy()

        idx = I.sample_sites(dims, n_even=n_even, n_rand=n_rand)
        cols = []
        xs = []
        for j, b in enumerate(sources()):
            t1 = time.time()
            x, it, res, st = oo.bicgstab(apply, b, tol, 2000)
            dt = time.time() - t1
            cols.append({"column": j, "iters": int(it), "true_resid": float(res), "status": int(st), "x_norm": float(np.linalg.norm(x)),
                         "oracle_solve_s": dt})
            xs.append(x[idx])
            print(f"[{name}] column {j}: iters {it} resid {res:.3e} status {st} in {dt:.0f} s", flush=True)
    rec = {"dims": list(dims), "kappa": kappa, "tol": tol, "plaquette": plaq, "u0": u0, "columns": cols,
           "sample": {"n_even": n_even, "n_rand": n_rand, "count": int(len(idx))},
           "oracle": {"workers": workers, "host_cores": os.cpu_count(), "stored_W": bool(store_W), "precalc_s": t_pre,
                      "applies": napply[0], "wall_s": time.time() - t0}}
    G.clear()
    return rec, np.stack(xs, axis=1)          # [sites, columns, 12]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", default="cfg2,cfg3,cfg4")
    ap.add_argument("--workers", type=int, default=os.cpu_count())
    args = ap.parse_args()
    D20, D32 = (20, 20, 20, 64), (32, 32, 32, 64)
    cases = {
        "cfg2": dict(dims=D20, links=lambda: I.near_identity_links(D20, 0.25, 5), kappa=0.10, tol=1e-6, store_W=True,
                     sources=lambda: [I.gaussian_spinor(D20, 6)], n_even=384, n_rand=384),
        "cfg3": dict(dims=D20, links=lambda: I.near_identity_links(D20, 0.25, 7), kappa=0.10, tol=1e-6, store_W=True,
                     sources=lambda: (I.point_source(D20, site=0, comp=j) for j in range(12)), n_even=192, n_rand=192),
        "cfg4": dict(dims=D32, links=lambda: I.haar_links(D32, 8), kappa=0.08, tol=1e-6, store_W=False,
                     sources=lambda: [I.gaussian_spinor(D32, 9)], n_even=256, n_rand=256),
    }
    jpath, zpath = os.path.join(HERE, "fullsize_bicgstab.json"), os.path.join(HERE, "fullsize_x_samples.npz")
    rec = json.load(open(jpath)) if os.path.exists(jpath) else {}
    xs = dict(np.load(zpath)) if os.path.exists(zpath) else {}
    for name in args.cases.split(","):
        r, x = run_case(name, workers=args.workers, **cases[name])
        rec[name], xs[name] = r, x
        json.dump(rec, open(jpath, "w"), indent=1, sort_keys=True)
        np.savez_compressed(zpath, **xs)
        print(f"[{name}] written", flush=True)


if __name__ == "__main__":
    main()
