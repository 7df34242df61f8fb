"""paper_2604_11920_b200 — thin Python binding of libtomolsqr.so (include/tomo_lsqr.h).

Argument marshalling only: every step of the hot path (CSR->CSC transpose, A v, A^T u, norms, scalar
recurrences, x/w update, stopping tests) runs in the library's CUDA kernels.  PyTorch supplies device
memory and streams.  There is NO fallback: if the shared library is missing or was not built, importing
the entry points raises.  Functions carry the names of the C ABI; :class:`TomoLsqr` is a convenience
wrapper that keeps the borrowed CSR tensors alive.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtomolsqr.so")

TOMO_OK = 0
TOMO_ERR_INVALID_ARG, TOMO_ERR_BAD_CSR, TOMO_ERR_NOT_DEVICE_PTR, TOMO_ERR_OOM = 1, 2, 3, 4
TOMO_ERR_CUDA, TOMO_ERR_UNSUPPORTED_ARCH, TOMO_ERR_RANGE, TOMO_ERR_NOALLOC_LIMIT = 5, 6, 7, 8
TOMO_NOALLOC_MAX_ROWS, TOMO_NOALLOC_MAX_SMS = 524288, 256   # include/tomo_lsqr.h
TOMO_VAL_F64, TOMO_VAL_F32 = 0, 1

# every symbol include/tomo_lsqr.h declares
SYMBOLS = (
    "tomo_lsqr_create", "tomo_lsqr_create_factored", "tomo_lsqr_assemble_csr", "tomo_lsqr_update_kernels", "tomo_lsqr_set_nodal_kernels", "tomo_lsqr_solve", "tomo_lsmr_solve", "tomo_lsqr_solve_host", "tomo_lsmr_solve_host",
    "tomo_lsqr_solve_multi", "tomo_lsmr_solve_multi", "tomo_lsqr_spmv", "tomo_lsqr_update_values", "tomo_lsqr_solve_sharded",
    "tomo_lsqr_get_csc", "tomo_lsqr_set_option", "tomo_lsqr_get_info", "tomo_lsqr_spmv_noalloc", "tomo_lsqr_destroy", "tomo_status_string",
)


# int allgather(void* ctx, const void* d_send, void* d_recv, size_t bytes, void* cuda_stream)
ALLGATHER_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)


class tomo_lsqr_result_t(ctypes.Structure):
    _fields_ = [("itn", ctypes.c_int32), ("istop", ctypes.c_int32), ("r1norm", ctypes.c_double),
                ("r2norm", ctypes.c_double), ("arnorm", ctypes.c_double), ("anorm", ctypes.c_double),
                ("acond", ctypes.c_double), ("xnorm", ctypes.c_double)]


class TomoError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status} ({tomo_status_string(status)})")


_lib = None


def load() -> ctypes.CDLL:
    """dlopen libtomolsqr.so (built in-tree by paper_2604_11920_b200.build); no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2604_11920_b200.build` "
                          "(CUDA library for sm_100a; there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, f64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_int
    lib.tomo_lsqr_create.argtypes = [ctypes.POINTER(vp), i64, i64, i64, vp, vp, vp, ci, vp]
    lib.tomo_lsqr_create_factored.argtypes = [ctypes.POINTER(vp), i64, i32, i64, i32, vp, vp, vp, i32, vp, vp, i64, i64, vp, vp, vp, vp]
    lib.tomo_lsqr_assemble_csr.argtypes = [i64, i32, i64, i32, vp, vp, vp, i32, vp, vp, i64, i64, vp, vp, vp, i64, vp, vp, vp, i32, vp]
    lib.tomo_lsqr_update_kernels.argtypes = [vp, vp, vp, vp]
    lib.tomo_lsqr_set_nodal_kernels.argtypes = [vp, vp, vp, vp]
    lib.tomo_lsqr_solve.argtypes = [vp, vp, f64, f64, f64, i32, vp, ctypes.POINTER(tomo_lsqr_result_t), vp, vp, vp]
    lib.tomo_lsmr_solve.argtypes = lib.tomo_lsqr_solve.argtypes
    lib.tomo_lsqr_solve_host.argtypes = [vp, vp, f64, f64, f64, i32, vp, ctypes.POINTER(tomo_lsqr_result_t), vp]
    lib.tomo_lsmr_solve_host.argtypes = lib.tomo_lsqr_solve_host.argtypes
    lib.tomo_lsqr_solve_multi.argtypes = [vp, i32, vp, f64, f64, f64, i32, vp, ctypes.POINTER(tomo_lsqr_result_t), vp]
    lib.tomo_lsmr_solve_multi.argtypes = lib.tomo_lsqr_solve_multi.argtypes
    lib.tomo_lsqr_spmv.argtypes = [vp, ci, vp, vp, vp]
    lib.tomo_lsqr_update_values.argtypes = [vp, vp, vp]
    lib.tomo_lsqr_solve_sharded.argtypes = [ctypes.POINTER(vp), i32, i32, i32, ALLGATHER_FN, vp, ctypes.POINTER(vp), f64, f64, f64, i32, vp,
                                            ctypes.POINTER(tomo_lsqr_result_t), vp]
    lib.tomo_lsqr_get_csc.argtypes = [vp, vp, vp, vp, vp]
    lib.tomo_lsqr_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    lib.tomo_lsqr_get_info.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(f64)]
    lib.tomo_lsqr_spmv_noalloc.argtypes = [i64, i64, i64, vp, vp, vp, ci, ci, vp, vp, vp]
    lib.tomo_lsqr_destroy.argtypes = [vp]
    lib.tomo_lsqr_destroy.restype = None
    lib.tomo_status_string.argtypes = [ci]
    lib.tomo_status_string.restype = ctypes.c_char_p
    for name in SYMBOLS:
        if name not in ("tomo_lsqr_destroy", "tomo_status_string"):
            getattr(lib, name).restype = ci
    _lib = lib
    return lib


def _ptr(t) -> int | None:
    """torch tensor / numpy array / int address / None -> address."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream) -> int | None:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    return getattr(stream, "cuda_stream", stream) or None


def tomo_status_string(status: int) -> str:
    return load().tomo_status_string(int(status)).decode()


def tomo_lsqr_create(m, n, nnz, d_rowptr, d_colind, d_vals, vt=TOMO_VAL_F64, stream=None) -> int:
    h = ctypes.c_void_p()
    st = load().tomo_lsqr_create(ctypes.byref(h), m, n, nnz, _ptr(d_rowptr), _ptr(d_colind), _ptr(d_vals), vt, _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_create")
    return h.value


def tomo_lsqr_create_factored(npairs, nper, nnodes, nz, d_lptr, d_lnode, d_lw, klen, d_kj0, d_kern, ms=0, snnz=0,
                              d_sptr=None, d_sidx=None, d_svals=None, stream=None) -> int:
    h = ctypes.c_void_p()
    st = load().tomo_lsqr_create_factored(ctypes.byref(h), int(npairs), int(nper), int(nnodes), int(nz), _ptr(d_lptr), _ptr(d_lnode),
                                          _ptr(d_lw), int(klen), _ptr(d_kj0), _ptr(d_kern), int(ms), int(snnz), _ptr(d_sptr),
                                          _ptr(d_sidx), _ptr(d_svals), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_create_factored")
    return h.value


def tomo_lsqr_assemble_csr(npairs, nper, nnodes, nz, d_lptr, d_lnode, d_lw, klen, d_kj0, d_kern, ms, snnz, d_sptr, d_sidx, d_svals,
                           nnz, d_rowptr, d_colind, d_vals, stream=None, nodal=0) -> None:
    """The factored description multiplied out into CSR device arrays (on-device assembly of G).  nodal=1: a kernel table per node."""
    st = load().tomo_lsqr_assemble_csr(int(npairs), int(nper), int(nnodes), int(nz), _ptr(d_lptr), _ptr(d_lnode), _ptr(d_lw), int(klen),
                                       _ptr(d_kj0), _ptr(d_kern), int(ms), int(snnz), _ptr(d_sptr), _ptr(d_sidx), _ptr(d_svals),
                                       int(nnz), _ptr(d_rowptr), _ptr(d_colind), _ptr(d_vals), int(nodal), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_assemble_csr")


def tomo_lsqr_update_kernels(h, d_kj0, d_kern, stream=None) -> None:
    st = load().tomo_lsqr_update_kernels(h, _ptr(d_kj0), _ptr(d_kern), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_update_kernels")


def tomo_lsqr_set_nodal_kernels(h, d_kj0, d_kern, stream=None) -> None:
    st = load().tomo_lsqr_set_nodal_kernels(h, _ptr(d_kj0), _ptr(d_kern), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_set_nodal_kernels")


def tomo_lsqr_destroy(h) -> None:
    if h:
        load().tomo_lsqr_destroy(h)


def tomo_lsqr_solve(h, d_b, damp, atol, btol, max_iters, d_x, h_r2norm_hist=None, h_arnorm_hist=None, stream=None) -> tomo_lsqr_result_t:
    res = tomo_lsqr_result_t()
    st = load().tomo_lsqr_solve(h, _ptr(d_b), damp, atol, btol, max_iters, _ptr(d_x), ctypes.byref(res),
                                _ptr(h_r2norm_hist), _ptr(h_arnorm_hist), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_solve")
    return res


def tomo_lsmr_solve(h, d_b, damp, atol, btol, max_iters, d_x, h_normr_hist=None, h_normar_hist=None, stream=None) -> tomo_lsqr_result_t:
    res = tomo_lsqr_result_t()
    st = load().tomo_lsmr_solve(h, _ptr(d_b), damp, atol, btol, max_iters, _ptr(d_x), ctypes.byref(res),
                                _ptr(h_normr_hist), _ptr(h_normar_hist), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsmr_solve")
    return res


def tomo_lsqr_solve_host(h, h_b, damp, atol, btol, max_iters, h_x, stream=None) -> tomo_lsqr_result_t:
    res = tomo_lsqr_result_t()
    st = load().tomo_lsqr_solve_host(h, _ptr(h_b), damp, atol, btol, max_iters, _ptr(h_x), ctypes.byref(res), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_solve_host")
    return res


def tomo_lsmr_solve_host(h, h_b, damp, atol, btol, max_iters, h_x, stream=None) -> tomo_lsqr_result_t:
    res = tomo_lsqr_result_t()
    st = load().tomo_lsmr_solve_host(h, _ptr(h_b), damp, atol, btol, max_iters, _ptr(h_x), ctypes.byref(res), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsmr_solve_host")
    return res


def tomo_lsqr_solve_multi(h, nrhs, d_B, damp, atol, btol, max_iters, d_X, stream=None):
    res = (tomo_lsqr_result_t * nrhs)()
    st = load().tomo_lsqr_solve_multi(h, nrhs, _ptr(d_B), damp, atol, btol, max_iters, _ptr(d_X), res, _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_solve_multi")
    return list(res)


def tomo_lsmr_solve_multi(h, nrhs, d_B, damp, atol, btol, max_iters, d_X, stream=None):
    res = (tomo_lsqr_result_t * nrhs)()
    st = load().tomo_lsmr_solve_multi(h, nrhs, _ptr(d_B), damp, atol, btol, max_iters, _ptr(d_X), res, _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsmr_solve_multi")
    return list(res)


def tomo_lsqr_spmv(h, transpose, d_in, d_out, stream=None) -> None:
    st = load().tomo_lsqr_spmv(h, int(transpose), _ptr(d_in), _ptr(d_out), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_spmv")


def tomo_lsqr_spmv_noalloc(m, n, nnz, d_rowptr, d_colind, d_vals, vt, accumulate, d_x, d_y, stream=None) -> None:
    """d_y <- A d_x over the caller's CSR without a handle and without any allocation (static scratch array in the library)."""
    st = load().tomo_lsqr_spmv_noalloc(int(m), int(n), int(nnz), _ptr(d_rowptr), _ptr(d_colind), _ptr(d_vals), int(vt), int(accumulate),
                                  _ptr(d_x), _ptr(d_y), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_spmv_noalloc")


class _RawBytes:
    """A raw device buffer (address, length) as a CUDA-array-interface object, so that torch can wrap it without a copy."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def make_allgather(dist, world_size: int, device: str = "cuda"):
    """The exchange of tomo_lsqr_solve_sharded on top of torch.distributed (marshalling only): wraps the two raw
    buffers the library hands over as byte tensors and calls all_gather_into_tensor (NCCL on `cuda`; `cpu` wraps host
    memory for the gloo test of this wrapper).  Returns the ctypes callback; keep a reference while it is in use."""
    import torch

    def wrap(ptr, nbytes):
        if device == "cuda":
            return torch.as_tensor(_RawBytes(ptr, nbytes), device="cuda")
        import numpy as np
        return torch.from_numpy(np.ctypeslib.as_array(ctypes.cast(ptr, ctypes.POINTER(ctypes.c_uint8)), shape=(nbytes,)))

    def allgather(ctx, d_send, d_recv, nbytes, stream):
        try:
            send, recv = wrap(d_send, nbytes), wrap(d_recv, nbytes * world_size)
            if device == "cuda":
                ext = torch.cuda.ExternalStream(stream) if stream else torch.cuda.default_stream()
                with torch.cuda.stream(ext):
                    dist.all_gather_into_tensor(recv, send)
            else:
                dist.all_gather_into_tensor(recv, send)
            return 0
        except Exception:  # noqa: BLE001 - a C callback must not raise
            return 1

    return ALLGATHER_FN(allgather)


def tomo_lsqr_solve_sharded(handles, d_bs, damp, atol, btol, max_iters, d_x, rank=0, nranks=1, allgather=None, stream=None) -> tomo_lsqr_result_t:
    """handles / d_bs: this rank's row blocks and their right-hand sides, in order; allgather: make_allgather(...) if nranks > 1."""
    nl = len(handles)
    hs = (ctypes.c_void_p * nl)(*handles)
    bs = (ctypes.c_void_p * nl)(*[_ptr(b) for b in d_bs])
    res = tomo_lsqr_result_t()
    cb = allgather if allgather is not None else ctypes.cast(None, ALLGATHER_FN)
    st = load().tomo_lsqr_solve_sharded(hs, nl, rank, nranks, cb, None, bs, damp, atol, btol, max_iters, _ptr(d_x), ctypes.byref(res),
                                        _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_solve_sharded")
    return res


def tomo_lsqr_update_values(h, d_vals, stream=None) -> None:
    st = load().tomo_lsqr_update_values(h, _ptr(d_vals), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_update_values")


def tomo_lsqr_get_csc(h, d_colptr, d_rowind, d_cvals, stream=None) -> None:
    st = load().tomo_lsqr_get_csc(h, _ptr(d_colptr), _ptr(d_rowind), _ptr(d_cvals), _stream(stream))
    if st != TOMO_OK:
        raise TomoError(st, "tomo_lsqr_get_csc")


def tomo_lsqr_set_option(h, key: str, value: int) -> None:
    st = load().tomo_lsqr_set_option(h, key.encode(), int(value))
    if st != TOMO_OK:
        raise TomoError(st, f"tomo_lsqr_set_option({key})")


def tomo_lsqr_get_info(h, key: str) -> float:
    out = ctypes.c_double()
    st = load().tomo_lsqr_get_info(h, key.encode(), ctypes.byref(out))
    if st != TOMO_OK:
        raise TomoError(st, f"tomo_lsqr_get_info({key})")
    return out.value


@dataclass
class Result:
    itn: int
    istop: int
    r1norm: float
    r2norm: float
    arnorm: float
    anorm: float
    acond: float
    xnorm: float

    @classmethod
    def of(cls, r: tomo_lsqr_result_t) -> "Result":
        return cls(r.itn, r.istop, r.r1norm, r.r2norm, r.arnorm, r.anorm, r.acond, r.xnorm)


class TomoLsqr:
    """Owns a handle and keeps the borrowed CSR device tensors alive (marshalling only)."""

    def __init__(self, m, n, rowptr, colind, vals, stream=None):
        import torch
        assert rowptr.is_cuda and colind.is_cuda and vals.is_cuda
        assert rowptr.dtype == torch.int64 and colind.dtype == torch.int32 and vals.dtype in (torch.float64, torch.float32)
        self.m, self.n, self.nnz = int(m), int(n), int(colind.numel())
        self._keep = (rowptr.contiguous(), colind.contiguous(), vals.contiguous())
        vt = TOMO_VAL_F64 if vals.dtype == torch.float64 else TOMO_VAL_F32
        self.h = tomo_lsqr_create(self.m, self.n, self.nnz, *self._keep, vt, stream)

    @classmethod
    def factored(cls, npairs, nper, nnodes, nz, lptr, lnode, lw, kj0, kern, sptr=None, sidx=None, svals=None, stream=None):
        """A handle on the factored operator (tomo_lsqr_create_factored); keeps the borrowed device tensors alive."""
        self = cls.__new__(cls)
        klen = int(kern.numel()) // int(nper)
        ms = 0 if sptr is None else int(sptr.numel()) - 1
        snnz = 0 if sidx is None else int(sidx.numel())
        keep = [None if t is None else t.contiguous() for t in (lptr, lnode, lw, kj0, kern, sptr, sidx, svals)]
        self._keep = tuple(keep)
        self.m, self.n = int(npairs) * int(nper) + ms, int(nnodes) * int(nz)
        self.nnz = int(lnode.numel()) * int(nper) * klen + snnz
        self.h = tomo_lsqr_create_factored(npairs, nper, nnodes, nz, keep[0], keep[1], keep[2], klen, keep[3], keep[4], ms, snnz,
                                           keep[5], keep[6], keep[7], stream)
        return self

    def set(self, **opts):
        for k, v in opts.items():
            tomo_lsqr_set_option(self.h, k, v)
        return self

    def info(self, key):
        return tomo_lsqr_get_info(self.h, key)

    def spmv(self, x, transpose=False):
        import torch
        out = torch.empty(self.n if transpose else self.m, dtype=torch.float64, device=x.device)
        tomo_lsqr_spmv(self.h, transpose, x, out)
        return out

    def update_values(self, vals):
        """New values on the same pattern (CSR order); the tensor replaces the borrowed value array."""
        assert vals.is_cuda and vals.dtype == self._keep[2].dtype and vals.numel() == self.nnz
        vals = vals.contiguous()
        tomo_lsqr_update_values(self.h, vals)
        self._keep = (self._keep[0], self._keep[1], vals)

    def csc(self):
        import torch
        dev = self._keep[0].device
        colptr = torch.empty(self.n + 1, dtype=torch.int64, device=dev)
        rowind = torch.empty(self.nnz, dtype=torch.int32, device=dev)
        cvals = torch.empty(self.nnz, dtype=self._keep[2].dtype, device=dev)
        tomo_lsqr_get_csc(self.h, colptr, rowind, cvals)
        return colptr, rowind, cvals

    def solve(self, b, damp=0.0, atol=0.0, btol=0.0, max_iters=50, history=False, solver="lsqr"):
        import numpy as np
        import torch
        x = torch.empty(self.n, dtype=torch.float64, device=b.device)
        r2 = np.full(max(max_iters, 1), np.nan) if history else None
        ar = np.full(max(max_iters, 1), np.nan) if history else None
        fn = {"lsqr": tomo_lsqr_solve, "lsmr": tomo_lsmr_solve}[solver]
        res = Result.of(fn(self.h, b, damp, atol, btol, max_iters, x, r2, ar))
        if history:
            return x, res, r2[: res.itn], ar[: res.itn]
        return x, res

    def solve_multi(self, B, damp=0.0, atol=0.0, btol=0.0, max_iters=50, solver="lsqr"):
        import torch
        nrhs = B.shape[1]
        X = torch.empty((self.n, nrhs), dtype=torch.float64, device=B.device)
        fn = {"lsqr": tomo_lsqr_solve_multi, "lsmr": tomo_lsmr_solve_multi}[solver]
        res = fn(self.h, nrhs, B.contiguous(), damp, atol, btol, max_iters, X)
        return X, [Result.of(r) for r in res]

    def close(self):
        if getattr(self, "h", None):
            tomo_lsqr_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
