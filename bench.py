#!/usr/bin/env python
"""bench.py -- the driver's benchmark contract for the OK-action hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A *step* is one pass of the whole hot path over one synthetic gauge
configuration of BASELINE.json configs[2] (20^3 x 64, fp32 W and spinors, eps = 0.25 links seed 5,
Gaussian source seed 6, kappa = 0.10, u0 = plaq^(1/4)):

    ok_precalc_W (a1+a2)  ->  NAPPLY x ok_dirac_apply (a3)  ->  ok_bicgstab to 1e-6 (a3+a4+a5)

`value` is BASELINE.json's metric: the Dirac apply's algorithmic HBM bandwidth, i.e.
(31 296 B/site x sites) / (mean device time of one ok_dirac_apply launch), measured with CUDA
events on the library's stream around the NAPPLY back-to-back applies of every timed step.
The W field (15.9 GB) is far larger than the 126 MB L2, so no flush is needed between launches.
The BiCGStab solve time, iteration count and the precalc time are reported beside it.

N > 1 (torchrun): the path does not shard in this build ("replicas only"): every rank
runs the same workload on its own GPU; `value` is the sum of the ranks' bytes over the max time.

--impl reference: the CPU oracle (oracle/ok_oracle.py, numpy fp64, as it stands) timed on the
host cores on a bounded sample of the same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1311_5029_b200 import inputs as I  # noqa: E402

METRIC = "OK Dirac apply HBM GB/s (% of B200 peak) + BiCGStab solve s at 20^3x64 fp32"
KERNEL_NAME = {(4, 1): "okd::apply_direct_kernel<float,...>", (8, 1): "okd::apply_direct_kernel<double,...>",
               (4, 12): "okd::apply_mrhs_kernel (tcgen05 kind::f16, both operands pre-split fp16 in HBM)"}
FLOP_PER_SITE = 27 * 144 * 8                                                             # 31 104
NAPPLY = 20

WORKLOADS = {
    # name: (dims, precision bytes, eps (None = Haar links), link seed, source seed, kappa, tol)
    "20x20x20x64-fp32": ((20, 20, 20, 64), 4, 0.25, 5, 6, 0.10, 1e-6),      # BASELINE configs[2] (the metric's config)
    "8x8x8x16-fp64": ((8, 8, 8, 16), 8, 0.30, 3, 2, 0.10, 1e-12),           # configs[1] shape, for quick runs
    "4x4x4x8-fp64": ((4, 4, 4, 8), 8, 0.30, 1, 2, 0.10, 1e-10),             # configs[0]
    "20x20x20x64-fp64": ((20, 20, 20, 64), 8, 0.25, 5, 6, 0.10, 1e-10),     # configs[2] lattice in fp64 (31.9 GB of W)
    "20x20x20x64-fp32-rhs12": ((20, 20, 20, 64), 4, 0.25, 7, None, 0.10, 1e-6),   # configs[3]: 12 point sources at the origin
    "32x32x32x64-fp32": ((32, 32, 32, 64), 4, None, 8, 9, 0.08, 1e-6),      # configs[4]: Haar links, 65 GB of W
    "4x4x4x8-fp32-rhs12": ((4, 4, 4, 8), 4, 0.25, 7, None, 0.10, 1e-6),     # quick check of the 12-RHS mode
}
NRHS = {"20x20x20x64-fp32-rhs12": 12, "4x4x4x8-fp32-rhs12": 12}
# reduced W storage: same lattice, links, source as configs[2]
WORKLOADS["20x20x20x64-fp32-block"] = WORKLOADS["20x20x20x64-fp32"]
WORKLOADS["20x20x20x64-fp32-ds"] = WORKLOADS["20x20x20x64-fp32"]
WORKLOADS["20x20x20x64-fp64-ds"] = WORKLOADS["20x20x20x64-fp64"]
WORKLOADS["32x32x32x64-fp32-ds"] = WORKLOADS["32x32x32x64-fp32"]
WORKLOADS["20x20x20x64-fp32-conj"] = WORKLOADS["20x20x20x64-fp32"]
WORKLOADS["20x20x20x64-fp64-conj"] = WORKLOADS["20x20x20x64-fp64"]
WORKLOADS["20x20x20x64-fp32-pauli"] = WORKLOADS["20x20x20x64-fp32"]
WORKLOADS["20x20x20x64-fp64-pauli"] = WORKLOADS["20x20x20x64-fp64"]
WORKLOADS["32x32x32x64-fp32-pauli"] = WORKLOADS["32x32x32x64-fp32"]
STORAGE = {"20x20x20x64-fp32-pauli": 4, "20x20x20x64-fp64-pauli": 4, "32x32x32x64-fp32-pauli": 4, "20x20x20x64-fp32-conj": 3, "20x20x20x64-fp64-conj": 3, "20x20x20x64-fp32-block": 1, "20x20x20x64-fp32-ds": 2, "20x20x20x64-fp64-ds": 2, "32x32x32x64-fp32-ds": 2}
W_COMPLEX_PER_SITE = {0: 27 * 144, 1: 260 * 9, 2: 132 * 9, 3: 70 * 9, 4: 37 * 9}


def make_links(dims, eps, lseed):
    return I.haar_links(dims, lseed) if eps is None else I.near_identity_links(dims, eps, lseed)


def alg_bytes_per_site(sbytes, nrhs, storage=0):
    """W once (in its storage format) + the spinor block read once + written once."""
    return W_COMPLEX_PER_SITE[storage] * 2 * sbytes + 2 * 24 * sbytes * nrhs


def fallback_peaks():
    return {"hbm_gbs": 6650.0, "_source": "fallback (B200_PROFILING.md)"}


def measured_peaks():
    try:
        d = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        d["_source"] = "measured (MEASURED_PEAKS.json)"
        return d
    except Exception:
        return fallback_peaks()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def __enter__(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None
        return self

    def __exit__(self, *a):
        if self.p:
            time.sleep(0.25)
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()

    def summary(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        try:
            self.f.flush()
            rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
            os.unlink(self.f.name)
            sm = [float(r[0]) for r in rows]
            out["samples"] = len(rows)
            if sm:
                out["sm_mhz"] = float(np.median(sm))
                out["sm_max_mhz"] = float(rows[0][1])
                out["power_w_max"] = max(float(r[2]) for r in rows)
                names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
                out["reasons"] = [n for k, n in enumerate(names) if any(r[3 + k].strip() == "Active" for r in rows)]
        except Exception as e:  # pragma: no cover
            out["error"] = str(e)
        return out


# ------------------------------------------------------------------------------ oracle arm
# The CPU baseline is the oracle AS IT STANDS (numpy fp64, oracle/ok_oracle.py); nothing in it is tuned for this.  The
# all-core leg only runs Oracle.apply_W on disjoint site ranges in forked worker processes (the sum over the 27 terms of a
# site never crosses a range) -- no change to the oracle's arithmetic.
_CPU = {}      # worker globals, inherited by fork
_ORACLE_SETUP = {}


def _cpu_worker(a, b, reps):
    o, psi, W, idx = _CPU["o"], _CPU["psi"], _CPU["W"], _CPU["idx"]
    for _ in range(reps):
        for col in psi:
            o.apply_W(col, idx=idx[a:b], W=W[a:b])
    return b - a


def oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=10.0, nsample=4096, U=None, nrhs=1, workers=1):
    """Times the oracle's stored-W apply (Eq. 2.2) on a bounded sample of the workload's sites, on `workers`
    host cores.  Returns dict(value = GB/s-equivalent of the fp32 contract bytes, cores, sample, ...)."""
    from oracle.ok_oracle import Oracle   # test infrastructure; allowed here for the CPU baseline only
    if U is None:
        U = make_links(dims, eps, lseed)
    key = (tuple(dims), id(U), kappa, nrhs, nsample, workers)
    if key not in _ORACLE_SETUP:     # the oracle object, the source columns and the sample's stored W are set up once per run
        u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
        o = Oracle(U, I.make_params(dims, kappa, u0))
        # the apply's cost is data-independent: Gaussian columns stand in for the point sources of the 12-RHS config
        cols = [I.gaussian_spinor(dims, (sseed if sseed is not None else 6) + j) for j in range(nrhs)]
        ns = min(nsample * workers, o.V)
        idx = (np.arange(ns) * (o.V // ns)).astype(np.int64)      # evenly spread sites
        t0 = time.perf_counter()
        W = o.precalc_W(idx)
        _ORACLE_SETUP[key] = (o, cols, ns, idx, W, time.perf_counter() - t0)
    o, cols, nsample, idx, W, t_pre = _ORACLE_SETUP[key]
    V = o.V
    reps = 0
    if workers == 1:
        c0, w0 = time.process_time(), time.perf_counter()
        while True:
            for psi in cols:
                o.apply_W(psi, idx=idx, W=W)
            reps += 1
            if time.perf_counter() - w0 > budget_s:
                break
        wall = time.perf_counter() - w0
        cores = max(1, int(round((time.process_time() - c0) / wall)))
    else:
        import multiprocessing as mp
        _CPU.update(o=o, psi=cols, W=W, idx=idx)
        step = (nsample + workers - 1) // workers
        chunks = [(a, min(nsample, a + step)) for a in range(0, nsample, step)]
        with mp.get_context("fork").Pool(workers) as pool:
            pool.starmap(_cpu_worker, [(a, b, 1) for a, b in chunks])          # warm the workers
            w0 = time.perf_counter()
            pool.starmap(_cpu_worker, [(a, b, 1) for a, b in chunks])
            one = time.perf_counter() - w0
            per = max(1, int(budget_s / max(one, 1e-3)))
            w0 = time.perf_counter()
            pool.starmap(_cpu_worker, [(a, b, per) for a, b in chunks])
            wall = time.perf_counter() - w0
            reps = per
        _CPU.clear()
        cores = workers
    sites_per_s = reps * nsample / wall
    return {"value": sites_per_s * alg_bytes_per_site(4, nrhs) / 1e9, "unit": "GB/s", "cores": cores,
            "kind": "oracle", "host_cores": os.cpu_count(),
            "sample": f"{nsample} evenly spaced sites of the {'x'.join(map(str, dims))} lattice, stored fp64 W, "
                      f"{reps} applies{' of %d columns' % nrhs if nrhs > 1 else ''} in {wall:.1f} s (numpy einsum"
                      f"{', %d forked workers over site ranges' % workers if workers > 1 else ''}); "
                      f"oracle precalc of the sample took {t_pre:.1f} s",
            "sites_per_s": sites_per_s, "applies_per_s_equiv": sites_per_s / V,
            "precalc_sites_per_s": nsample / t_pre}


def oracle_direct_vs_W(dims=(8, 8, 8, 16)):
    """The paper's "Naive" (gauge-link products every apply) against its "Precalc" (stored W) inverter, in the oracle's own
    terms: one Oracle.apply_direct and repeated Oracle.apply_W on the whole 8^3 x 16 lattice of BASELINE configs[1]
    (Table 1a at PAPER.md:130-135), one core."""
    from oracle.ok_oracle import Oracle
    U = I.near_identity_links(dims, 0.3, 3)
    o = Oracle(U, I.make_params(dims, 0.10, I.tadpole_u0(I.mean_plaquette(dims, U))))
    psi = I.gaussian_spinor(dims, 2)
    t0 = time.perf_counter()
    a = o.apply_direct(psi)
    t_direct = time.perf_counter() - t0
    t0 = time.perf_counter()
    W = o.precalc_W()
    t_pre = time.perf_counter() - t0
    t_w = []
    for _ in range(3):
        t0 = time.perf_counter()
        b = o.apply_W(psi, W=W)
        t_w.append(time.perf_counter() - t0)
    t_W = float(np.median(t_w))
    return {"lattice": "x".join(map(str, dims)), "cores": 1, "apply_direct_s": t_direct, "apply_W_s": t_W, "precalc_W_s": t_pre,
            "direct_over_W": t_direct / t_W, "forms_agree_rel_l2": float(np.linalg.norm(a - b) / np.linalg.norm(b)),
            "what": "oracle.apply_direct (link products, the paper's 'Naive') vs oracle.apply_W (Eq. 2.2 with stored W, 'Precalc')"}


PAPER_CONTEXT = {
    "source": "PAPER.md:120-122, Table 1 (PAPER.md:130-146); context, not the target",
    "hardware": "MILC coarse 20^3x64 lattice on 4 nodes of the SNU cluster DAVID1, each node one core of an Intel i7-920 + one NVIDIA GTX480 "
                "(1.5 GB), single-rail QLogic InfiniBand",
    "precalculation_speedup_vs_naive": 3.9, "cuda_speedup_vs_naive": 13.1, "cuda_speedup_vs_precalc_cpu": 3.4,
    "total_cg_time_s": {"naive": 11814.8, "precalc": 3046.6, "cuda": 898.7},
    "dirac_multiply_ms_per_iteration_sp_dp": {"cpu_precalc": [962, 1206], "cuda_kernel_only": [32, 107]},
    "gtx480_gflops": {"multiply_only": 58.7, "with_host_copies": 18.2},
}


def cpu_baseline_legs(dims, eps, lseed, sseed, kappa, U, nrhs):
    """the oracle's stored-W apply at ONE core and at ALL host cores, and its direct form once."""
    ncore = os.cpu_count() or 1
    one = oracle_sample(dims, eps, lseed, sseed, kappa, U=U, nrhs=nrhs, nsample=4096 if nrhs == 1 else 512, budget_s=8.0)
    allc = oracle_sample(dims, eps, lseed, sseed, kappa, U=U, nrhs=nrhs, nsample=2048 if nrhs == 1 else 256, budget_s=8.0, workers=ncore) \
        if ncore > 1 else dict(one)
    allc["one_core"] = {k: one[k] for k in ("value", "unit", "cores", "sample", "sites_per_s", "applies_per_s_equiv")}
    allc["all_over_one_core"] = allc["value"] / one["value"]
    allc["direct_form"] = oracle_direct_vs_W()
    return allc


def run_reference(args, wl):
    dims, sbytes, eps, lseed, sseed, kappa, tol = WORKLOADS[wl]
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    U = make_links(dims, eps, lseed)
    nrhs = NRHS.get(wl, 1)
    ncore = os.cpu_count() or 1
    per = []
    for _ in range(args.warmup):
        oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=1.0, nsample=256, U=U, nrhs=nrhs, workers=ncore)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        per.append(oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=4.0, nsample=512, U=U, nrhs=nrhs, workers=ncore))
    wall = time.perf_counter() - t0
    val = float(np.mean([p["value"] for p in per]))
    cb = dict(per[-1])
    cb["value"] = val
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl, "note": "CPU oracle on all host cores, bounded sample of the workload's sites per step"},
            "cpu_baseline": cb, "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "paper_context": PAPER_CONTEXT}
    print(json.dumps(line))


# ------------------------------------------------------------------------------ our arm
def max_over_ranks(values, dist, device):
    """Replicas-only aggregation: every rank times the same workload on its own GPU;
    the job's time is the slowest rank's.  `dist` is torch.distributed (initialised) or None."""
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_value(world, alg_bytes, apply_ms):
    """Whole-job GB/s of `world` replicas that each moved alg_bytes in apply_ms (max over ranks)."""
    return world * alg_bytes / (apply_ms * 1e-3) / 1e9


KERNEL_SOURCE = {"dense1": "ok_apply.cu", "mrhs": "ok_apply_mrhs.cu", "sparse": "ok_apply_sparse.cu"}
GOLDEN_CASE = {"20x20x20x64-fp32": "cfg2", "20x20x20x64-fp32-rhs12": "cfg3", "32x32x32x64-fp32": "cfg4"}


def source_sha16(name):
    import hashlib
    try:
        return hashlib.sha256(open(os.path.join(ROOT, "paper_1311_5029_b200", "csrc", name), "rb").read()).hexdigest()[:16]
    except OSError:
        return None


def ncu_record(wl):
    """The committed ncu --set full capture of this workload's apply kernel (profiles/apply_ncu_traffic.csv): DRAM bytes per
    launch and, for the 12-RHS mode, the tensor-pipe counter.  The row names the kernel's source file and its sha256 at capture
    time; if the file has changed since, the numbers are withheld (traffic = null) and the record says so."""
    import csv
    try:
        rows = [r for r in csv.DictReader(open(os.path.join(ROOT, "profiles", "apply_ncu_traffic.csv"))) if r["workload"] == wl]
    except Exception:
        rows = []
    if not rows:
        return {"traffic": None, "traffic_source": None}
    r = rows[-1]
    now = source_sha16(r["kernel_source"])
    out = {"traffic_source": r["source"], "traffic_kernel_source": "paper_1311_5029_b200/csrc/" + r["kernel_source"],
           "traffic_kernel_sha": r["kernel_source_sha16"], "kernel_sha_now": now, "traffic_stale": now != r["kernel_source_sha16"]}
    if out["traffic_stale"]:
        out["traffic"] = None
        return out
    out["traffic"] = int(r["dram_bytes_per_launch"])
    out["ncu_dram_cycles_active_pct"] = float(r["dram_cycles_active_pct"]) if r.get("dram_cycles_active_pct") else None
    out["ncu_tensor_pipe_active_pct"] = float(r["tensor_pipe_active_pct"]) if r.get("tensor_pipe_active_pct") else None
    return out


def oracle_golden(wl):
    """Iteration count / true residual of the ORACLE's own BiCGStab on this workload (tests/golden/fullsize_bicgstab.json, written
    by tests/golden/make_fullsize_golden.py from oracle/ only) -- printed beside the CUDA path's (north_star: within +-2)."""
    case = GOLDEN_CASE.get(wl)
    try:
        g = json.load(open(os.path.join(ROOT, "tests", "golden", "fullsize_bicgstab.json")))[case]
        return {"iters": max(c["iters"] for c in g["columns"]), "true_resid": max(c["true_resid"] for c in g["columns"]),
                "source": "tests/golden/fullsize_bicgstab.json[%s]" % case}
    except Exception:
        return None


class Prepared:
    """One workload resident in HBM: links, W, workspace, packed source and result vectors."""

    def __init__(self, wl, dev, stream, U=None):
        import torch
        from paper_1311_5029_b200 import binding as B
        self.wl, self.dev, self.stream = wl, dev, stream
        self.dims, self.sbytes, eps, lseed, sseed, self.kappa, self.tol = WORKLOADS[wl]
        self.nrhs = NRHS.get(wl, 1)
        self.storage = STORAGE.get(wl, 0)
        self.U = make_links(self.dims, eps, lseed) if U is None else U
        self.plaq = I.mean_plaquette(self.dims, self.U)
        self.pd = I.make_params(self.dims, self.kappa, I.tadpole_u0(self.plaq))
        self.p = B.make_params(self.pd, B.OK_FP32 if self.sbytes == 4 else B.OK_FP64, nrhs=self.nrhs, storage=self.storage)
        self.V = int(np.prod(self.dims))
        self.cdt = torch.complex64 if self.sbytes == 4 else torch.complex128
        if self.nrhs == 1:
            self.psi_np = I.gaussian_spinor(self.dims, sseed)
        else:      # configs[3]: all 12 spin-colour point sources at the origin, canonical [site][comp][rhs]
            self.psi_np = np.stack([I.point_source(self.dims, site=0, comp=j) for j in range(self.nrhs)], axis=2)
        self.links = torch.from_numpy(self.U).to(dev)
        canon = torch.from_numpy(self.psi_np).to(self.cdt).to(dev)
        self.W = B.alloc_W(self.p, dev)
        self.work = B.alloc_work(self.p, dev)
        self.src, self.out, self.x = B.alloc_vec(self.p, dev), B.alloc_vec(self.p, dev), B.alloc_vec(self.p, dev)
        B.ok_set_stream(stream)
        B.ok_set_workspace(self.work)
        with torch.cuda.stream(stream):
            B.ok_pack_spinor(self.p, canon, self.src)
        stream.synchronize()
        self.alg = self.V * alg_bytes_per_site(self.sbytes, self.nrhs, self.storage)
        self.kernel = (KERNEL_NAME[(self.sbytes, self.nrhs)] if self.storage == 0 else
                       ("okd::apply_pauli_kernel<%s>" % ("float" if self.sbytes == 4 else "double")) if self.storage == 4 else
                       "okd::apply_sparse_kernel<%s,%d>" % ("float" if self.sbytes == 4 else "double", self.storage))

    def step(self, rec=None):
        """precalc + NAPPLY applies + solve; CUDA-event times of the three parts appended to rec."""
        import torch
        from paper_1311_5029_b200 import binding as B
        st = self.stream
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        with torch.cuda.stream(st):
            ev[0].record(st)
            B.ok_precalc_W(self.links, self.p, self.W)
            ev[1].record(st)
            for _ in range(NAPPLY):
                B.ok_dirac_apply(self.W, self.src, self.out)
            ev[2].record(st)
            status, it, res = B.ok_bicgstab(self.W, self.src, self.x, self.tol, 5000, raise_on_fail=False)
            ev[3].record(st)
        if status != 0:
            raise RuntimeError(f"ok_bicgstab failed: {B.ok_strerror(status)}")
        if rec is not None:
            st.synchronize()
            rec["pre_ms"].append(ev[0].elapsed_time(ev[1]))
            rec["apply_ms"].append(ev[1].elapsed_time(ev[2]) / NAPPLY)
            rec["solve_s"].append(ev[2].elapsed_time(ev[3]) / 1e3)
            rec["iters"].append(it)
            rec["resid"].append(res)

    def timed(self, steps, warmup, index, barrier):
        import torch
        from paper_1311_5029_b200 import binding as B
        rec = {"pre_ms": [], "apply_ms": [], "solve_s": [], "iters": [], "resid": []}
        for _ in range(warmup):
            self.step(None)
        barrier()
        l0 = B.ok_launch_count()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(index) as cs:
            t0.record(self.stream)
            for _ in range(steps):
                self.step(rec)
            t1.record(self.stream)
            barrier()
        rec["total_ms"] = t0.elapsed_time(t1)
        rec["launches"] = B.ok_launch_count() - l0
        rec["clocks"] = cs.summary()
        return rec

    def many_applies(self, n, index):
        """n back-to-back ok_dirac_apply, each bracketed by CUDA events on the library's stream (BASELINE configs[2]: 1000 timed
        applies; median and min of the per-apply times)."""
        import torch
        from paper_1311_5029_b200 import binding as B
        st = self.stream
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        with ClockSampler(index) as cs:
            with torch.cuda.stream(st):
                for _ in range(20):
                    B.ok_dirac_apply(self.W, self.src, self.out)
                ev[0].record(st)
                for k in range(n):
                    B.ok_dirac_apply(self.W, self.src, self.out)
                    ev[k + 1].record(st)
            st.synchronize()
        ms = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(n)])
        gb = self.alg / 1e6
        return {"n": n, "warmup": 20, "ms_mean": float(ms.mean()), "ms_median": float(np.median(ms)), "ms_min": float(ms.min()),
                "ms_max": float(ms.max()), "GBps_mean": gb / float(ms.mean()), "GBps_median": gb / float(np.median(ms)),
                "GBps_best": gb / float(ms.min()), "total_ms": ev[0].elapsed_time(ev[n]), "clocks": cs.summary()}

    def roofline(self, a_ms, peaks):
        ach = self.alg / (a_ms * 1e-3) / 1e9
        r = {"bound": "hbm", "kernel": self.kernel, "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
             "frac_of_nominal_8000": ach / 8000.0, "peak_source": peaks["_source"], "algorithmic_bytes_per_launch": self.alg}
        r.update(ncu_record(self.wl))
        if self.storage == 4:
            # OK_W_PAULI is bound by the fp32 pipes, not by HBM: 68 matrix uses x 36 complex MACs x 8 flop per site
            # against 148 SMs x 128 lanes x 2 flop x sm_max_mhz; the HBM figures above stay for comparison with the other formats
            flops = 68 * 36 * 8 * self.V
            peak = 148 * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
            r["alu"] = {"bound": "alu", "achieved": flops / (a_ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                        "frac": flops / (a_ms * 1e-3) / 1e12 / peak, "flops_per_launch": flops,
                        "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 flop x sm_max_mhz (DESIGN.md 6.6)"}
        return r

    def tensor(self, a_ms, clocks, peaks, ncu):
        # per site 21 tcgen05.mma of M = 128, N = 48, K = 16 (24 cycles each on one SM's tensor pipe, measured); useful flops are the
        # complex contraction's
        sm_mhz = clocks.get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
        return {"kind": "tcgen05.mma.kind::f16 (fp16 hi/lo split of fp32 operands), fp32 accumulate in TMEM", "mma_per_site": 21,
                "mma_shape": [128, 48, 16], "pipe_busy_frac_from_cycles": 21 * 24 * (self.V / 148.0) / (a_ms * 1e-3 * sm_mhz * 1e6),
                "ncu_sm__pipe_tensor_cycles_active_pct": ncu.get("ncu_tensor_pipe_active_pct"), "ncu_source": ncu.get("traffic_source"),
                "issued_tflops": self.V * 21 * 2 * 128 * 48 * 16 / (a_ms * 1e-3) / 1e12,
                "useful_tflops": self.V * FLOP_PER_SITE * self.nrhs / (a_ms * 1e-3) / 1e12,
                "note": "the mode is HBM-bound (W streams once for 12 columns)"}

    def release(self):
        import torch
        from paper_1311_5029_b200 import binding as B
        B.ok_set_workspace(None)
        B.ok_forget_W(self.W)
        self.W = self.work = self.src = self.out = self.x = self.links = None
        torch.cuda.empty_cache()


def sub_record(wl, dev, stream, index, peaks, steps=2):
    """One BASELINE config as a sub-record of the default line: same step, its own roofline, clocks and CUDA-event times."""
    P = Prepared(wl, dev, stream)
    rec = P.timed(steps, 3, index, lambda: stream.synchronize())
    a_ms = float(np.mean(rec["apply_ms"]))
    roof = P.roofline(a_ms, peaks)
    out = {"workload": wl, "dtype": "f32" if P.sbytes == 4 else "f64", "nrhs": P.nrhs, "sites": P.V, "steps": steps, "warmup": 3,
           "step": f"ok_precalc_W + {NAPPLY} x ok_dirac_apply + ok_bicgstab(tol={P.tol:g})", "W_GB": P.alg / 1e9,
           "apply_ms": a_ms, "value": roof["achieved"], "unit": "GB/s", "applies_per_s": 1e3 / a_ms,
           "gflops": P.V * FLOP_PER_SITE * P.nrhs / (a_ms * 1e-3) / 1e9,
           "bicgstab_solve_s": float(np.mean(rec["solve_s"])), "bicgstab_iters": int(np.max(rec["iters"])),
           "bicgstab_true_resid": float(np.max(rec["resid"])), "bicgstab_tol": P.tol, "oracle_bicgstab": oracle_golden(wl),
           "precalc_ms": float(np.mean(rec["pre_ms"])), "ms_per_step": rec["total_ms"] / steps, "roofline": roof,
           "gpu_launches": int(rec["launches"]), "clocks": rec["clocks"], "plaquette": P.plaq, "u0": P.pd["u0"]}
    if P.nrhs == 12:
        out["tensor"] = P.tensor(a_ms, rec["clocks"], peaks, roof)
    P.release()
    return out


def slab_record(wl, nslab, dev, stream, index, peaks, steps=2):
    """The t-slab decomposition (ok_slab_* in include/ok.h) on ONE GPU: the lattice of workload wl cut into nslab
    slabs held by this process (virtual ranks: separate W and fields per slab; the applies read the neighbours' boundary
    slices in place, ok_slab_dirac_apply_peer, as they would read a peer GPU's mapped memory), so
    that the cost of the decomposition itself -- the extra launches, the halo loads, the per-slab reduction stage -- is
    measured against the unsharded numbers.  No inter-GPU transfer is involved or claimed."""
    import torch
    from paper_1311_5029_b200 import binding as B
    from paper_1311_5029_b200 import slab as S
    dims, sbytes, eps, lseed, sseed, kappa, tol = WORKLOADS[wl]
    U = make_links(dims, eps, lseed)
    plaq = I.mean_plaquette(dims, U)
    pd = I.make_params(dims, kappa, I.tadpole_u0(plaq))
    p = B.make_params(pd, B.OK_FP32 if sbytes == 4 else B.OK_FP64)
    ranges = S.slab_ranges(dims[3], nslab)
    slab = B.make_slab_params(p, ranges[0][1])
    plocal = B.make_params(dict(pd, dims=tuple(dims[:3]) + (ranges[0][1],)), p.precision)
    cdt = torch.complex64 if sbytes == 4 else torch.complex128
    work = B.alloc_bytes(B.ok_slab_work_bytes(slab, nslab, 1), dev)
    B.ok_set_stream(stream)
    B.ok_set_workspace(work, work.numel())
    psi = I.gaussian_spinor(dims, sseed)
    Ws, links, src, out, xs = [], [], [], [], []
    for t0, Tl in ranges:
        Ws.append(B.alloc_W(slab, dev))
        links.append(torch.from_numpy(S.link_window(U, dims, t0, Tl)).to(dev))
        v = torch.zeros(B.ok_slab_vec_bytes(slab), dtype=torch.uint8, device=dev)
        with torch.cuda.stream(stream):
            B.ok_pack_spinor(plocal, torch.from_numpy(S.spinor_slab(psi, dims, t0, Tl)).to(cdt).to(dev), S.interior(slab, v))
        src.append(v)
        out.append(torch.zeros_like(v))
        xs.append(torch.zeros_like(v))
    stream.synchronize()
    V = int(np.prod(dims))
    rec = {"pre_ms": [], "apply_ms": [], "solve_s": [], "iters": [], "resid": []}
    # (lower neighbour's last own slice, upper neighbour's first own slice) of every slab
    faces = [(S.halo_views(slab, src[(i - 1) % nslab])[2], S.halo_views(slab, src[(i + 1) % nslab])[1]) for i in range(nslab)]

    def step(record):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            for (t0, Tl), W, lk in zip(ranges, Ws, links):
                B.ok_slab_precalc_W(lk, slab, dims[3], t0, W)
            ev[1].record(stream)
            for _ in range(NAPPLY):
                for i in range(nslab):       # the neighbours' boundary slices are read in place (what ok_slab_bicgstab does internally)
                    B.ok_slab_dirac_apply_peer(Ws[i], src[i], faces[i][0], faces[i][1], out[i])
            ev[2].record(stream)
            st, it, res = B.ok_slab_bicgstab(Ws, src, xs, tol, 5000, raise_on_fail=False)
            ev[3].record(stream)
        if st != 0:
            raise RuntimeError(f"ok_slab_bicgstab failed: {B.ok_strerror(st)}")
        if record:
            stream.synchronize()
            rec["pre_ms"].append(ev[0].elapsed_time(ev[1]))
            rec["apply_ms"].append(ev[1].elapsed_time(ev[2]) / NAPPLY)
            rec["solve_s"].append(ev[2].elapsed_time(ev[3]) / 1e3)
            rec["iters"].append(it)
            rec["resid"].append(res)

    for _ in range(3):
        step(False)
    stream.synchronize()
    l0 = B.ok_launch_count()
    with ClockSampler(index) as cs:
        for _ in range(steps):
            step(True)
        stream.synchronize()
    a_ms = float(np.mean(rec["apply_ms"]))
    alg = V * alg_bytes_per_site(sbytes, 1, 0)
    ach = alg / (a_ms * 1e-3) / 1e9
    outrec = {"workload": wl, "slabs": nslab, "Tloc": ranges[0][1], "what": "t-slab decomposition on one GPU (virtual ranks; halo exchange fused into the apply: neighbours' boundary slices read in place)",
              "apply_ms": a_ms, "value": ach, "unit": "GB/s", "halo_bytes_per_apply_per_slab": 2 * B.ok_slab_slice_bytes(slab),
              "bicgstab_solve_s": float(np.mean(rec["solve_s"])), "bicgstab_iters": int(np.max(rec["iters"])),
              "bicgstab_true_resid": float(np.max(rec["resid"])), "bicgstab_tol": tol, "oracle_bicgstab": oracle_golden(wl),
              "precalc_ms": float(np.mean(rec["pre_ms"])),
              "roofline": {"bound": "hbm", "kernel": "okd::apply_direct_kernel<float,...> over %d slabs" % nslab, "achieved": ach, "peak": peaks["hbm_gbs"],
                           "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "peak_source": peaks["_source"], "algorithmic_bytes_per_launch": alg // nslab,
                           "traffic": None},
              "gpu_launches": int(B.ok_launch_count() - l0), "clocks": cs.summary(), "steps": steps, "warmup": 3}
    B.ok_set_workspace(None)
    for W in Ws:
        B.ok_forget_W(W)
    del Ws, links, src, out, xs, work
    torch.cuda.empty_cache()
    return outrec


def run_ours(args, wl):
    import torch
    from paper_1311_5029_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dims, sbytes, eps, lseed, sseed, kappa, tol = WORKLOADS[wl]
    nrhs = NRHS.get(wl, 1)
    # ---- inputs (seeded, synthetic; generated on the host) and the CPU baseline legs -- before CUDA is initialised, so that the
    #      all-core leg can fork worker processes safely
    U = make_links(dims, eps, lseed)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_legs(dims, eps, lseed, sseed, kappa, U, nrhs)
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the OK hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    B.lib()
    stream = torch.cuda.Stream(device=dev)
    P = Prepared(wl, dev, stream, U=U)      # resident in HBM before timing
    V, p, W = P.V, P.p, P.W

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    rec = P.timed(args.steps, max(args.warmup, 3), local, barrier)
    total_ms, launches, clocks = rec["total_ms"], rec["launches"], rec["clocks"]

    # ---- BASELINE configs[2]: 1000 timed applies (median / min / mean of the per-apply event times)
    many = P.many_applies(1000 if V >= 100000 else 200, local) if not args.no_extras else None

    # ---- end to end through the host-buffer C-ABI call: pinned host psi -> H2D -> pack -> apply -> unpack -> D2H
    host_in = torch.from_numpy(P.psi_np).to(P.cdt).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    for _ in range(3):
        B.ok_dirac_apply_host(W, host_in, host_out)
    n_e2e = max(args.steps, 5)
    barrier()
    e0 = time.perf_counter()
    for _ in range(n_e2e):
        B.ok_dirac_apply_host(W, host_in, host_out)      # synchronises the stream itself
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - e0) / n_e2e
    io_bytes = V * 12 * 2 * sbytes * nrhs

    # ---- fp64 workloads: the mixed-precision inversion of the same system (both W sets resident), outside the timed steps
    mixed = None
    if sbytes == 8 and nrhs == 1:
        p32 = B.make_params(P.pd, B.OK_FP32, storage=P.storage)
        W32 = B.alloc_W(p32, dev)
        mwork = B.alloc_bytes(max(B.ok_mixed_work_bytes(p), B.ok_work_bytes(p32)), dev)
        B.ok_set_workspace(mwork)
        m_s = []
        with torch.cuda.stream(stream):
            B.ok_precalc_W(P.links, p32, W32)
            for _ in range(1 + max(args.steps, 3)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                mst, mit, mout, mres = B.ok_bicgstab_mixed(W, W32, P.src, P.x, tol, 1e-4, 5000, 50, raise_on_fail=False)
                e1.record(stream)
                stream.synchronize()
                m_s.append(e0.elapsed_time(e1) / 1e3)
        mixed = {"solve_s": float(np.mean(m_s[1:])), "status": mst, "inner_iters": mit, "outer": mout, "true_resid": mres,
                 "inner_tol": 1e-4, "what": "ok_bicgstab_mixed(W64, W32): fp32 BiCGStab inside fp64 defect correction, same tol"}
        B.ok_set_workspace(P.work)
        del W32, mwork

    # ---- max over ranks
    a_ms = float(np.mean(rec["apply_ms"]))
    total_ms, a_ms, e2e_ms, s_s = max_over_ranks([total_ms, a_ms, e2e_ms, float(np.mean(rec["solve_s"]))], dist, dev)
    alg = P.alg
    value = aggregate_value(world, alg, a_ms)
    peaks = measured_peaks()

    if rank == 0:
        roof = P.roofline(a_ms, peaks)
        line = {
            "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if sbytes == 4 else "f64", "data": "synthetic",
            "config": {"workload": wl, "nrhs": nrhs, "storage": ["dense", "block (260 colour blocks)", "ds (132 colour blocks)", "conj (70 colour blocks)", "pauli (49 colour blocks as 37 stored matrices)"][P.storage], "step": f"ok_precalc_W + {NAPPLY} x ok_dirac_apply + ok_bicgstab(tol={tol:g})",
                       "sites": V, "l2_flush": "not needed: W (%.1f GB) >> L2 (126 MB)" % (B.ok_W_bytes(p) / 1e9),
                       "parallelism": "replicas only" if world > 1 else "single GPU", "plaquette": P.plaq, "u0": P.pd["u0"]},
            "pct_of_peak": {"measured_copy": 100 * value / world / peaks["hbm_gbs"], "nominal_8000": 100 * value / world / 8000.0},
            "apply_ms": a_ms, "applies_per_s": world * 1e3 / a_ms, "sites_per_s": world * V * 1e3 / a_ms,
            "gflops": world * V * FLOP_PER_SITE * nrhs / (a_ms * 1e-3) / 1e9,
            "bicgstab_solve_s": s_s, "bicgstab_iters": int(np.max(rec["iters"])), "bicgstab_true_resid": float(np.max(rec["resid"])),
            "bicgstab_tol": tol, "oracle_bicgstab": oracle_golden(wl),
            "precalc_ms": float(np.mean(rec["pre_ms"])),
            "roofline": roof,
            "e2e": {"value": world * alg / (e2e_ms * 1e-3) / 1e9, "unit": "GB/s", "ms_per_apply": e2e_ms,
                    "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "what": "ok_dirac_apply_host: pinned host psi -> device, pack, apply, unpack, -> pinned host; W resident"},
            "gpu_launches": int(launches), "clocks": clocks, "paper_context": PAPER_CONTEXT,
        }
        if many is not None:
            line["applies_1000"] = many
        if nrhs == 12:
            line["tensor"] = P.tensor(a_ms, clocks, peaks, roof)
        if mixed is not None:
            line["mixed_precision"] = mixed
        if cpu is not None:
            line["cpu_baseline"] = cpu
        # ---- the other BASELINE configs as sub-records of the default line (single GPU, default workload only)
        if world == 1 and wl == "20x20x20x64-fp32" and not args.no_extras:
            del host_in, host_out
            P.release()
            line["configs"] = {}
            for name, sub in [("configs[3] 12 RHS", "20x20x20x64-fp32-rhs12"), ("configs[2] lattice in fp64", "20x20x20x64-fp64"),
                              ("configs[4] 32^3x64 Haar", "32x32x32x64-fp32"),
                              ("configs[2] in the paper's 50-colour-block compression (OK_W_PAULI)", "20x20x20x64-fp32-pauli")]:
                try:
                    line["configs"][name] = sub_record(sub, dev, stream, local, peaks)
                except Exception as e:      # a sub-record must not take the contract line down with it
                    line["configs"][name] = {"workload": sub, "error": repr(e)[:300]}
            try:
                line["configs"]["configs[2] as 4 t-slabs (one GPU)"] = slab_record("20x20x20x64-fp32", 4, dev, stream, local, peaks)
            except Exception as e:
                line["configs"]["configs[2] as 4 t-slabs (one GPU)"] = {"error": repr(e)[:300]}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: apply-throughput sweep over lattice sizes (Haar links seed 8, kappa 0.08, fp32), single GPU.
    One JSON line: per lattice and W storage format the mean device time of an ok_dirac_apply and the derived rates."""
    import torch
    from paper_1311_5029_b200 import binding as B
    dev = "cuda:0"
    torch.cuda.set_device(0)
    B.lib()
    stream = torch.cuda.Stream(device=dev)
    B.ok_set_stream(stream)
    rows = []
    for dims in [(8, 8, 8, 16), (12, 12, 12, 24), (16, 16, 16, 32), (20, 20, 20, 64), (24, 24, 24, 64), (32, 32, 32, 64)]:
        U = I.haar_links(dims, 8)
        pd = I.make_params(dims, 0.08, I.tadpole_u0(I.mean_plaquette(dims, U)))
        links = torch.from_numpy(U).to(dev)
        V = int(np.prod(dims))
        psi = torch.from_numpy(I.gaussian_spinor(dims, 9)).to(torch.complex64).to(dev)
        for storage in (0, 2, 3, 4):
            p = B.make_params(pd, B.OK_FP32, storage=storage)
            W, work = B.alloc_W(p, dev), B.alloc_work(p, dev)
            src, out = B.alloc_vec(p, dev), B.alloc_vec(p, dev)
            B.ok_set_workspace(work)
            with torch.cuda.stream(stream):
                B.ok_precalc_W(links, p, W)
                B.ok_pack_spinor(p, psi, src)
                for _ in range(5):
                    B.ok_dirac_apply(W, src, out)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                nrep = 200 if V < 200000 else 50
                e0.record(stream)
                for _ in range(nrep):
                    B.ok_dirac_apply(W, src, out)
                e1.record(stream)
            stream.synchronize()
            ms = e0.elapsed_time(e1) / nrep
            alg = V * alg_bytes_per_site(4, 1, storage)
            rows.append({"dims": "x".join(map(str, dims)), "sites": V, "storage": ["dense", "block", "ds", "conj", "pauli"][storage],
                         "W_GB": B.ok_W_bytes(p) / 1e9, "apply_ms": ms, "GBps": alg / ms / 1e6, "sites_per_s": V / ms * 1e3,
                         "gflops": V * FLOP_PER_SITE / ms / 1e6})
            B.ok_set_workspace(None)
            B.ok_forget_W(W)
            del W, work, src, out
        del links, psi
    print(json.dumps({"metric": "OK Dirac apply throughput sweep (fp32, Haar links seed 8, kappa 0.08)", "n_gpus": 1, "sweep": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="20x20x20x64-fp32", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the 1000-apply series and the sub-records of the other BASELINE configs")
    ap.add_argument("--slabs", type=int, default=0, help="time the t-slab decomposition of the workload with this many slabs on one GPU")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: apply throughput over lattice sizes (not the driver's contract line)")
    args = ap.parse_args()
    if args.slabs:
        import torch
        from paper_1311_5029_b200 import binding as B
        torch.cuda.set_device(0)
        B.lib()
        print(json.dumps(slab_record(args.workload, args.slabs, "cuda:0", torch.cuda.Stream(device="cuda:0"), 0, measured_peaks(), steps=args.steps)))
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, args.workload)
    else:
        run_ours(args, args.workload)


if __name__ == "__main__":
    main()
