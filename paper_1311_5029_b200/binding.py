"""Thin ctypes binding of libokdirac (include/ok.h): same names, argument marshalling only.

Every step of the hot path runs inside the CUDA library.  PyTorch is used for device memory
(torch tensors own every buffer) and streams.  If ``libokdirac.so`` is missing, or a call
returns an error status, an exception is raised -- there is no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os

OK_FP32, OK_FP64 = 0, 1
OK_W_DENSE, OK_W_BLOCK, OK_W_DS, OK_W_CONJ, OK_W_PAULI = 0, 1, 2, 3, 4
OK_NTERMS = 27
OK_W_HEADER_BYTES = 1024
OK_SLAB, OK_SLAB_LINK_HALO = 1, 2

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libokdirac.so")
_lib = None


class OkError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: status {status}: {ok_strerror(status)}")


class ok_params(C.Structure):
    _fields_ = [("dims", C.c_int32 * 4), ("precision", C.c_int32), ("bc", C.c_int32 * 4), ("nrhs", C.c_int32),
                ("kappa", C.c_double), ("u0", C.c_double), ("zeta", C.c_double), ("rs", C.c_double),
                ("cB", C.c_double), ("cE", C.c_double), ("cEE", C.c_double), ("c1", C.c_double),
                ("c2", C.c_double), ("c3", C.c_double), ("c4", C.c_double), ("c5", C.c_double),
                ("storage", C.c_int32), ("reserved_", C.c_int32)]


EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t)
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int)


BARRIER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p)


class ok_slab_peers(C.Structure):
    _fields_ = [("lo_work", C.c_void_p), ("hi_work", C.c_void_p), ("lo_x", C.c_void_p), ("hi_x", C.c_void_p), ("barrier", BARRIER_FN),
                ("user", C.c_void_p)]


class ok_comm(C.Structure):
    _fields_ = [("rank", C.c_int32), ("nranks", C.c_int32), ("exchange", EXCHANGE_FN), ("allgather", ALLGATHER_FN), ("user", C.c_void_p)]


EXPORTS = {
    # name: (restype, argtypes)
    "ok_W_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_vec_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_work_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_set_stream": (C.c_int, [C.c_void_p]),
    "ok_set_workspace": (C.c_int, [C.c_void_p, C.c_size_t]),
    "ok_pack_spinor": (C.c_int, [C.POINTER(ok_params), C.c_void_p, C.c_void_p]),
    "ok_unpack_spinor": (C.c_int, [C.POINTER(ok_params), C.c_void_p, C.c_void_p]),
    "ok_pack_W": (C.c_int, [C.POINTER(ok_params), C.c_void_p, C.c_void_p]),
    "ok_unpack_W": (C.c_int, [C.c_void_p, C.c_void_p]),
    "ok_precalc_W": (C.c_int, [C.c_void_p, C.POINTER(ok_params), C.c_void_p]),
    "ok_dirac_apply": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "ok_bicgstab": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int,
                              C.POINTER(C.c_int), C.POINTER(C.c_double)]),
    "ok_dirac_apply_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "ok_dirac_apply_dot_static": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "ok_static_max_sites": (C.c_size_t, []),
    "ok_static_strerror": (C.c_char_p, []),
    "ok_cgnr": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double)]),
    "ok_W_unit_index": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int)]),
    "ok_mixed_work_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_bicgstab_mixed": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int,
                                    C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_double)]),
    "ok_slab_slice_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_slab_vec_bytes": (C.c_size_t, [C.POINTER(ok_params)]),
    "ok_slab_work_bytes": (C.c_size_t, [C.POINTER(ok_params), C.c_int, C.c_int]),
    "ok_slab_precalc_W": (C.c_int, [C.c_void_p, C.POINTER(ok_params), C.c_int, C.c_int, C.c_void_p]),
    "ok_slab_dirac_apply": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "ok_slab_dirac_apply_peer": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "ok_slab_set_peers": (C.c_int, [C.POINTER(ok_slab_peers)]),
    "ok_slab_bicgstab": (C.c_int, [C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_double, C.c_int,
                                   C.POINTER(ok_comm), C.POINTER(C.c_int), C.POINTER(C.c_double)]),
    "ok_W_params": (C.c_int, [C.c_void_p, C.POINTER(ok_params)]),
    "ok_forget_W": (C.c_int, [C.c_void_p]),
    "ok_launch_count": (C.c_uint64, []),
    "ok_strerror": (C.c_char_p, [C.c_int]),
    "ok_version": (C.c_char_p, []),
}


def lib():
    """Load libokdirac.so (once).  Fails loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} not found: build it with `python -m paper_1311_5029_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array / int."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _check(status, where):
    if status != 0:
        raise OkError(status, where)


def make_params(p: dict, precision: int, nrhs: int = 1, storage: int = 0) -> ok_params:
    """dict (inputs.make_params) -> C struct."""
    q = ok_params()
    q.storage, q.reserved_ = storage, 0
    q.dims[:] = list(p["dims"])
    q.bc[:] = list(p["bc"])
    q.precision, q.nrhs = precision, nrhs
    for k in ("kappa", "u0", "zeta", "rs", "cB", "cE", "cEE", "c1", "c2", "c3", "c4", "c5"):
        setattr(q, k, float(p[k]))
    return q


# ------------------------------------------------------------------ same-name wrappers
def ok_strerror(status):
    return lib().ok_strerror(int(status)).decode()


def ok_version():
    return lib().ok_version().decode()


def ok_W_bytes(p):
    return lib().ok_W_bytes(C.byref(p))


def ok_vec_bytes(p):
    return lib().ok_vec_bytes(C.byref(p))


def ok_work_bytes(p):
    return lib().ok_work_bytes(C.byref(p))


def ok_set_stream(stream=None):
    """stream: torch.cuda.Stream, raw cudaStream_t int, or None (legacy default stream)."""
    h = 0 if stream is None else (stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))
    _check(lib().ok_set_stream(h), "ok_set_stream")


def ok_set_workspace(buf, nbytes=None):
    if buf is None:
        _check(lib().ok_set_workspace(None, 0), "ok_set_workspace")
        return
    n = nbytes if nbytes is not None else buf.numel() * buf.element_size()
    _check(lib().ok_set_workspace(_ptr(buf), n), "ok_set_workspace")


def ok_pack_spinor(p, canon, packed):
    _check(lib().ok_pack_spinor(C.byref(p), _ptr(canon), _ptr(packed)), "ok_pack_spinor")


def ok_unpack_spinor(p, packed, canon):
    _check(lib().ok_unpack_spinor(C.byref(p), _ptr(packed), _ptr(canon)), "ok_unpack_spinor")


def ok_pack_W(p, canon_W, W):
    _check(lib().ok_pack_W(C.byref(p), _ptr(canon_W), _ptr(W)), "ok_pack_W")


def ok_unpack_W(W, canon_W):
    _check(lib().ok_unpack_W(_ptr(W), _ptr(canon_W)), "ok_unpack_W")


def ok_precalc_W(links, p, W):
    _check(lib().ok_precalc_W(_ptr(links), C.byref(p), _ptr(W)), "ok_precalc_W")


def ok_dirac_apply(W, psi, out):
    _check(lib().ok_dirac_apply(_ptr(W), _ptr(psi), _ptr(out)), "ok_dirac_apply")


def ok_static_max_sites():
    return lib().ok_static_max_sites()


def ok_static_strerror():
    return lib().ok_static_strerror().decode()


def ok_dirac_apply_dot_static(W, psi, a, out, result):
    """out = M psi, result (device, 3 doubles) = Re<a,out>, Im<a,out>, ||out||^2; allocates nothing (ok.h)."""
    st = lib().ok_dirac_apply_dot_static(_ptr(W), _ptr(psi), _ptr(a), _ptr(out), _ptr(result))
    if st != 0:
        raise OkError(st, "ok_dirac_apply_dot_static: " + ok_static_strerror())


def ok_dirac_apply_host(W, psi_host, out_host):
    _check(lib().ok_dirac_apply_host(_ptr(W), _ptr(psi_host), _ptr(out_host)), "ok_dirac_apply_host")


def ok_bicgstab(W, src, x, tol, maxit, raise_on_fail=True):
    """Returns (status, iters, true_relative_residual)."""
    it, res = C.c_int(0), C.c_double(0.0)
    st = lib().ok_bicgstab(_ptr(W), _ptr(src), _ptr(x), float(tol), int(maxit), C.byref(it), C.byref(res))
    if st != 0 and raise_on_fail:
        raise OkError(st, "ok_bicgstab")
    return st, it.value, res.value


def ok_cgnr(W, src, x, tol, maxit, raise_on_fail=True):
    """Returns (status, iters, true_relative_residual)."""
    it, res = C.c_int(0), C.c_double(0.0)
    st = lib().ok_cgnr(_ptr(W), _ptr(src), _ptr(x), float(tol), int(maxit), C.byref(it), C.byref(res))
    if st != 0 and raise_on_fail:
        raise OkError(st, "ok_cgnr")
    return st, it.value, res.value


def ok_W_unit_index(storage, term, row, col):
    """Returns (unit, stored, sign, conj, shift_term); unit = -1 for a structural zero."""
    info = (C.c_int * 4)()
    u = lib().ok_W_unit_index(int(storage), int(term), int(row), int(col), info)
    return u, info[0], info[1], info[2], info[3]


def ok_mixed_work_bytes(p):
    return lib().ok_mixed_work_bytes(C.byref(p))


def ok_bicgstab_mixed(W64, W32, src, x, tol, inner_tol, maxit, max_outer=50, raise_on_fail=True):
    """Returns (status, inner_iters_total, outer_corrections, true_relative_residual)."""
    it, outer, res = C.c_int(0), C.c_int(0), C.c_double(0.0)
    st = lib().ok_bicgstab_mixed(_ptr(W64), _ptr(W32), _ptr(src), _ptr(x), float(tol), float(inner_tol), int(maxit), int(max_outer),
                                 C.byref(it), C.byref(outer), C.byref(res))
    if st != 0 and raise_on_fail:
        raise OkError(st, "ok_bicgstab_mixed")
    return st, it.value, outer.value, res.value


def make_slab_params(p: ok_params, Tloc: int) -> ok_params:
    """The parameters of a t-slab of Tloc time slices of the lattice p (ok.h: reserved_ = OK_SLAB, dims[3] = Tloc)."""
    q = ok_params.from_buffer_copy(bytes(p))
    q.dims[3] = int(Tloc)
    q.reserved_ = OK_SLAB
    return q


def ok_slab_slice_bytes(slab):
    return lib().ok_slab_slice_bytes(C.byref(slab))


def ok_slab_vec_bytes(slab):
    return lib().ok_slab_vec_bytes(C.byref(slab))


def ok_slab_work_bytes(slab, nslab=1, nranks=1):
    return lib().ok_slab_work_bytes(C.byref(slab), int(nslab), int(nranks))


def ok_slab_precalc_W(links_ext, slab, T_global, t0, W):
    _check(lib().ok_slab_precalc_W(_ptr(links_ext), C.byref(slab), int(T_global), int(t0), _ptr(W)), "ok_slab_precalc_W")


def ok_slab_dirac_apply(W, psi_ext, out_ext):
    _check(lib().ok_slab_dirac_apply(_ptr(W), _ptr(psi_ext), _ptr(out_ext)), "ok_slab_dirac_apply")


def ok_slab_dirac_apply_peer(W, psi_ext, lo_slice, hi_slice, out_ext):
    """lo_slice / hi_slice: device addresses (tensor views or ints) of the neighbours' boundary slices (ok.h)."""
    _check(lib().ok_slab_dirac_apply_peer(_ptr(W), _ptr(psi_ext), _ptr(lo_slice), _ptr(hi_slice), _ptr(out_ext)), "ok_slab_dirac_apply_peer")


def ok_slab_set_peers(peers):
    """peers: ok_slab_peers (keep it and its callback alive while set) or None to clear."""
    _check(lib().ok_slab_set_peers(C.byref(peers) if peers is not None else None), "ok_slab_set_peers")


def ok_slab_bicgstab(W, src_ext, x_ext, tol, maxit, comm=None, raise_on_fail=True):
    """W, src_ext, x_ext: lists (one entry per slab this process holds, in t order).  comm: ok_comm or None.
    Returns (status, iters, true_relative_residual)."""
    n = len(W)
    arr = lambda ts: (C.c_void_p * n)(*[_ptr(t) for t in ts])
    it, res = C.c_int(0), C.c_double(0.0)
    st = lib().ok_slab_bicgstab(n, arr(W), arr(src_ext), arr(x_ext), float(tol), int(maxit), C.byref(comm) if comm is not None else None,
                                C.byref(it), C.byref(res))
    if st != 0 and raise_on_fail:
        raise OkError(st, "ok_slab_bicgstab")
    return st, it.value, res.value


def ok_W_params(W):
    q = ok_params()
    _check(lib().ok_W_params(_ptr(W), C.byref(q)), "ok_W_params")
    return q


def ok_forget_W(W):
    _check(lib().ok_forget_W(_ptr(W)), "ok_forget_W")


def ok_launch_count():
    return int(lib().ok_launch_count())


# ------------------------------------------------------------------ device-memory helpers (torch)
def alloc_bytes(nbytes, device="cuda:0"):
    """Caller-owned device buffer (torch owns the memory; 256-byte aligned by the caching allocator)."""
    import torch
    return torch.empty(int(nbytes), dtype=torch.uint8, device=device)


def alloc_W(p, device="cuda:0"):
    """W buffer; the library's record of it is dropped when the tensor is freed (the caching
    allocator hands the same address out again, ok.h: ok_forget_W)."""
    import weakref
    t = alloc_bytes(ok_W_bytes(p), device)
    weakref.finalize(t, lib().ok_forget_W, t.data_ptr())
    return t


def alloc_vec(p, device="cuda:0"):
    return alloc_bytes(ok_vec_bytes(p), device)


def alloc_work(p, device="cuda:0"):
    return alloc_bytes(ok_work_bytes(p), device)
