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
               (4, 12): "okd::apply_mrhs_kernel (tcgen05 kind::f16, split fp16) + okd::colmax_kernel"}
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
STORAGE = {"20x20x20x64-fp32-conj": 3, "20x20x20x64-fp64-conj": 3, "20x20x20x64-fp32-block": 1, "20x20x20x64-fp32-ds": 2, "20x20x20x64-fp64-ds": 2, "32x32x32x64-fp32-ds": 2}
W_COMPLEX_PER_SITE = {0: 27 * 144, 1: 260 * 9, 2: 132 * 9, 3: 70 * 9}


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
def oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=12.0, nsample=4096, U=None, nrhs=1):
    """Times the oracle's stored-W apply (Eq. 2.2) on a bounded sample of the workload's sites.
    Returns dict(value GB/s-equivalent of the fp32 contract bytes, cores, sample, ...)."""
    from oracle.ok_oracle import Oracle   # test infrastructure; allowed here for the CPU baseline only
    if U is None:
        U = make_links(dims, eps, lseed)
    u0 = I.tadpole_u0(I.mean_plaquette(dims, U))
    o = Oracle(U, I.make_params(dims, kappa, u0))
    # the apply's cost is data-independent: Gaussian columns stand in for the point sources of the 12-RHS config
    cols = [I.gaussian_spinor(dims, (sseed if sseed is not None else 6) + j) for j in range(nrhs)]
    V = o.V
    nsample = min(nsample, V)
    idx = (np.arange(nsample) * (V // nsample)).astype(np.int64)      # evenly spread sites
    t0 = time.perf_counter()
    W = o.precalc_W(idx)
    t_pre = time.perf_counter() - t0
    c0, w0 = time.process_time(), time.perf_counter()
    reps = 0
    while True:
        for psi in cols:
            o.apply_W(psi, idx=idx, W=W)
        reps += 1
        if time.perf_counter() - w0 > budget_s:
            break
    wall = time.perf_counter() - w0
    cpu = time.process_time() - c0
    sites_per_s = reps * nsample / wall
    return {"value": sites_per_s * alg_bytes_per_site(4, nrhs) / 1e9, "unit": "GB/s", "cores": max(1, int(round(cpu / wall))),
            "kind": "oracle", "host_cores": os.cpu_count(),
            "sample": f"{nsample} evenly spaced sites of the {'x'.join(map(str, dims))} lattice, stored fp64 W, "
                      f"{reps} applies{' of %d columns' % nrhs if nrhs > 1 else ''} in {wall:.1f} s (numpy einsum); "
                      f"oracle precalc of the sample took {t_pre:.1f} s",
            "sites_per_s": sites_per_s, "applies_per_s_equiv": sites_per_s / V,
            "precalc_sites_per_s": nsample / t_pre}


def run_reference(args, wl):
    dims, sbytes, eps, lseed, sseed, kappa, tol = WORKLOADS[wl]
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    U = make_links(dims, eps, lseed)
    nrhs = NRHS.get(wl, 1)
    per = []
    for _ in range(args.warmup):
        oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=1.0, nsample=1024, U=U, nrhs=nrhs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        per.append(oracle_sample(dims, eps, lseed, sseed, kappa, budget_s=4.0, nsample=2048, U=U, nrhs=nrhs))
    wall = time.perf_counter() - t0
    val = float(np.mean([p["value"] for p in per]))
    cb = dict(per[-1])
    cb["value"] = val
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl, "note": "CPU oracle, bounded sample of the workload's sites per step"},
            "cpu_baseline": cb, "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
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


def run_ours(args, wl):
    import torch
    from paper_1311_5029_b200 import binding as B

    dims, sbytes, eps, lseed, sseed, kappa, tol = WORKLOADS[wl]
    prec = B.OK_FP32 if sbytes == 4 else B.OK_FP64
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the OK hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    B.lib()

    # ---- inputs (seeded, synthetic; generated on the host, resident in HBM before timing)
    nrhs = NRHS.get(wl, 1)
    U = make_links(dims, eps, lseed)
    plaq = I.mean_plaquette(dims, U)
    pd = I.make_params(dims, kappa, I.tadpole_u0(plaq))
    storage = STORAGE.get(wl, 0)
    p = B.make_params(pd, prec, nrhs=nrhs, storage=storage)
    V = int(np.prod(dims))
    cdt = torch.complex64 if sbytes == 4 else torch.complex128
    if nrhs == 1:
        psi_np = I.gaussian_spinor(dims, sseed)
    else:      # configs[3]: all 12 spin-colour point sources at the origin, canonical [site][comp][rhs]
        psi_np = np.stack([I.point_source(dims, site=0, comp=j) for j in range(nrhs)], axis=2)
    links = torch.from_numpy(U).to(dev)
    canon = torch.from_numpy(psi_np).to(cdt).to(dev)
    W = B.alloc_W(p, dev)
    work = B.alloc_work(p, dev)
    src, out, x = B.alloc_vec(p, dev), B.alloc_vec(p, dev), B.alloc_vec(p, dev)
    stream = torch.cuda.Stream(device=dev)
    B.ok_set_stream(stream)
    B.ok_set_workspace(work)
    with torch.cuda.stream(stream):
        B.ok_pack_spinor(p, canon, src)
    stream.synchronize()

    apply_ms, solve_s, pre_ms, iters_l, resid_l = [], [], [], [], []

    def step(record):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            B.ok_precalc_W(links, p, W)
            ev[1].record(stream)
            for _ in range(NAPPLY):
                B.ok_dirac_apply(W, src, out)
            ev[2].record(stream)
            st, it, res = B.ok_bicgstab(W, src, x, tol, 5000, raise_on_fail=False)
            ev[3].record(stream)
        if st != 0:
            raise RuntimeError(f"ok_bicgstab failed: {B.ok_strerror(st)}")
        if record:
            stream.synchronize()
            pre_ms.append(ev[0].elapsed_time(ev[1]))
            apply_ms.append(ev[1].elapsed_time(ev[2]) / NAPPLY)
            solve_s.append(ev[2].elapsed_time(ev[3]) / 1e3)
            iters_l.append(it)
            resid_l.append(res)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step(False)
    barrier()
    l0 = B.ok_launch_count()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as cs:
        t_start.record(stream)
        for _ in range(args.steps):
            step(True)
        t_end.record(stream)
        barrier()
    total_ms = t_start.elapsed_time(t_end)
    launches = B.ok_launch_count() - l0
    clocks = cs.summary()

    # ---- end to end through the host-buffer C-ABI call: pinned host psi -> H2D -> pack -> apply -> unpack -> D2H
    host_in = torch.from_numpy(psi_np).to(cdt).pin_memory()
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
        p32 = B.make_params(pd, B.OK_FP32, storage=storage)
        W32 = B.alloc_W(p32, dev)
        mwork = B.alloc_bytes(max(B.ok_mixed_work_bytes(p), B.ok_work_bytes(p32)), dev)
        B.ok_set_workspace(mwork)
        m_s = []
        with torch.cuda.stream(stream):
            B.ok_precalc_W(links, p32, W32)
            for _ in range(1 + max(args.steps, 3)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                mst, mit, mout, mres = B.ok_bicgstab_mixed(W, W32, src, x, tol, 1e-4, 5000, 50, raise_on_fail=False)
                e1.record(stream)
                stream.synchronize()
                m_s.append(e0.elapsed_time(e1) / 1e3)
        mixed = {"solve_s": float(np.mean(m_s[1:])), "status": mst, "inner_iters": mit, "outer": mout, "true_resid": mres,
                 "inner_tol": 1e-4, "what": "ok_bicgstab_mixed(W64, W32): fp32 BiCGStab inside fp64 defect correction, same tol"}
        B.ok_set_workspace(work)
        del W32, mwork

    # ---- max over ranks
    a_ms = float(np.mean(apply_ms))
    total_ms, a_ms, e2e_ms, s_s = max_over_ranks([total_ms, a_ms, e2e_ms, float(np.mean(solve_s))], dist, dev)
    alg = V * alg_bytes_per_site(sbytes, nrhs, storage)
    value = aggregate_value(world, alg, a_ms)
    peaks = measured_peaks()

    if rank == 0:
        traffic = None
        try:
            import csv
            for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "apply_ncu_traffic.csv"))):
                if row["workload"] == wl:      # ncu --set full capture of the same kernel, per launch
                    traffic = int(row["dram_bytes_per_launch"])
        except Exception:
            pass
        cpu = (oracle_sample(dims, eps, lseed, sseed, kappa, U=U, nrhs=nrhs, nsample=4096 if nrhs == 1 else 1024)
               if world == 1 and not args.no_cpu_baseline else None)
        line = {
            "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if sbytes == 4 else "f64", "data": "synthetic",
            "config": {"workload": wl, "nrhs": nrhs, "storage": ["dense", "block (260 colour blocks)", "ds (132 colour blocks)", "conj (70 colour blocks)"][storage], "step": f"ok_precalc_W + {NAPPLY} x ok_dirac_apply + ok_bicgstab(tol={tol:g})",
                       "sites": V, "l2_flush": "not needed: W (%.1f GB) >> L2 (126 MB)" % (B.ok_W_bytes(p) / 1e9),
                       "parallelism": "replicas only" if world > 1 else "single GPU", "plaquette": plaq, "u0": pd["u0"]},
            "pct_of_peak": {"measured_copy": 100 * value / world / peaks["hbm_gbs"], "nominal_8000": 100 * value / world / 8000.0},
            "apply_ms": a_ms, "applies_per_s": world * 1e3 / a_ms, "sites_per_s": world * V * 1e3 / a_ms,
            "gflops": world * V * FLOP_PER_SITE * nrhs / (a_ms * 1e-3) / 1e9,
            "bicgstab_solve_s": s_s, "bicgstab_iters": int(np.max(iters_l)), "bicgstab_true_resid": float(np.max(resid_l)),
            "precalc_ms": float(np.mean(pre_ms)),
            "roofline": {"bound": "hbm", "kernel": KERNEL_NAME[(sbytes, nrhs)] if storage == 0 else "okd::apply_sparse_kernel<%s,%d>" % ("float" if sbytes == 4 else "double", storage), "achieved": alg / (a_ms * 1e-3) / 1e9,
                         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": alg / (a_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                         "peak_source": peaks["_source"], "algorithmic_bytes_per_launch": alg, "traffic": traffic},
            "e2e": {"value": world * alg / (e2e_ms * 1e-3) / 1e9, "unit": "GB/s", "ms_per_apply": e2e_ms,
                    "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "what": "ok_dirac_apply_host: pinned host psi -> device, pack, apply, unpack, -> pinned host; W resident"},
            "gpu_launches": int(launches), "clocks": clocks,
        }
        if nrhs == 12:
            # tensor-pipe report for the multi-RHS mode (north_star): per site 21 tcgen05.mma of M=64, N=48, K=16 (24 cycles
            # each on one SM's tensor pipe, measured), i.e. 504 busy cycles per site; useful flops are the complex contraction's
            sm_mhz = clocks.get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
            busy = 21 * 24 * (V / 148.0) / (a_ms * 1e-3 * sm_mhz * 1e6)
            line["tensor"] = {"kind": "tcgen05.mma.kind::f16 (fp16 hi/lo split of fp32 operands), fp32 accumulate in TMEM",
                              "mma_per_site": 21, "mma_shape": [64, 48, 16], "pipe_busy_frac_est": busy,
                              "issued_tflops": world * V * 21 * 2 * 64 * 48 * 16 / (a_ms * 1e-3) / 1e12,
                              "useful_tflops": world * V * FLOP_PER_SITE * nrhs / (a_ms * 1e-3) / 1e12,
                              "note": "the mode is HBM-bound (W streams once for 12 columns); ncu sm__pipe_tensor_cycles_active: profiles/"}
        if mixed is not None:
            line["mixed_precision"] = mixed
        if cpu is not None:
            line["cpu_baseline"] = cpu
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
        for storage in (0, 2, 3):
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
            rows.append({"dims": "x".join(map(str, dims)), "sites": V, "storage": ["dense", "block", "ds", "conj"][storage],
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
    ap.add_argument("--sweep", action="store_true", help="configs[4]: apply throughput over lattice sizes (not the driver's contract line)")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, args.workload)
    else:
        run_ours(args, args.workload)


if __name__ == "__main__":
    main()
