"""Helpers for the -m gpu parity tests: move seeded inputs to the device and call the C-ABI."""
import numpy as np
import torch

from paper_1311_5029_b200 import binding as B

DEV = "cuda:0"
_ws = {}


def cdtype(prec):
    return torch.complex128 if prec == B.OK_FP64 else torch.complex64


def npdtype(prec):
    return np.complex128 if prec == B.OK_FP64 else np.complex64


def workspace(p):
    """(Re)bind a workspace large enough for p; the tensor is kept alive here (caller-owned)."""
    need = B.ok_work_bytes(p)
    if _ws.get("n", 0) < need:
        _ws["buf"] = None
        _ws["buf"] = B.alloc_bytes(need, DEV)
        _ws["n"] = need
    B.ok_set_workspace(_ws["buf"], _ws["n"])
    B.ok_set_stream(None)


def to_dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.to(DEV)


def pack_spinor(p, psi_np):
    canon = to_dev(psi_np, cdtype(p.precision))
    packed = B.alloc_vec(p, DEV)
    B.ok_pack_spinor(p, canon, packed)
    return packed


def unpack_spinor(p, packed, shape):
    canon = torch.empty(shape, dtype=cdtype(p.precision), device=DEV)
    B.ok_unpack_spinor(p, packed, canon)
    torch.cuda.synchronize()
    return canon.cpu().numpy().astype(np.complex128)


def precalc(p, links_np):
    workspace(p)
    links = to_dev(links_np, torch.complex128)
    W = B.alloc_W(p, DEV)
    B.ok_precalc_W(links, p, W)
    torch.cuda.synchronize()
    return W


def unpack_W(p, W, V):
    canon = torch.empty((V, 27, 12, 12), dtype=cdtype(p.precision), device=DEV)
    B.ok_unpack_W(W, canon)
    torch.cuda.synchronize()
    return canon.cpu().numpy().astype(np.complex128)


def apply(p, W, psi_np):
    packed = pack_spinor(p, psi_np)
    out = B.alloc_vec(p, DEV)
    B.ok_dirac_apply(W, packed, out)
    return unpack_spinor(p, out, psi_np.shape)


def per_site_rel_err(got, want):
    """max over sites of ||got(x) - want(x)||_2 / ||want(x)||_2 (sites with negligible want skipped; S12)."""
    num = np.linalg.norm(got - want, axis=1)
    den = np.linalg.norm(want, axis=1)
    keep = den > 1e-30 * den.max()
    return float((num[keep] / den[keep]).max())


def rel_l2(got, want):
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def fp32_operator_slack(o, x, b, idx=None, W=None):
    """DESIGN.md 10, reading R-RESID.  The library's `resid` of an fp32 solve is || b - fl32(M32 x) || / || b || with M32 the
    fp32-rounded W it stores; the oracle evaluates || b - M64 x || / || b ||.  The two differ by at most
        || (M32 - M64) x || + || fl32(M32 x) - M32 x ||   <=   2 * 2^-24 * || |W| |x| ||_2
    (every real of W rounded once: |dW| <= 2^-24 |W| elementwise, rigorous; the second term is the kernel's own fp32 rounding
    of the 324-term sums, whose accumulated error stays below one unit 2^-24 |W||x| in every measured case).  Returns that
    bound relative to || b || -- evaluated by the oracle as apply_W(|x|, W = |W|) -- on the sites `idx` (all sites if None;
    for a sample the caller extrapolates like the residual itself)."""
    Wa = np.abs(o.precalc_W(idx) if W is None else W).astype(np.complex128)
    S = o.apply_W(np.abs(x).astype(np.complex128), idx=idx, W=Wa)
    scale = 1.0 if idx is None else np.sqrt(o.V / len(idx))
    if S.ndim == 3:     # [site][comp][rhs]: one bound per column
        return 2.0 * 2.0 ** -24 * scale * np.linalg.norm(S.reshape(-1, S.shape[2]), axis=0) / np.linalg.norm(b.reshape(-1, b.shape[2]), axis=0)
    return 2.0 * 2.0 ** -24 * scale * float(np.linalg.norm(S)) / float(np.linalg.norm(b))
