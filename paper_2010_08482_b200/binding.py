"""ctypes binding of libctqmc_b200.so (include/ctqmc.h).  Argument marshalling only: every step of the path
(routing, chain product, rescaling, trace, norms) runs in the library's CUDA kernels.  There is no CPU fallback: if the
library cannot be loaded, importing this module's functions raises.

The function names are the C names.  Device arrays are torch CUDA tensors (torch is used for device memory and streams
only); host arrays are numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libctqmc_b200.so")

CTQMC_OK, CTQMC_ERR_ARG, CTQMC_ERR_OOM, CTQMC_ERR_CUDA, CTQMC_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
CTQMC_STATUS_OK, CTQMC_STATUS_VANISHING, CTQMC_STATUS_INVALID = 0, 1, 2
CTQMC_SCHEDULE_THIN, CTQMC_SCHEDULE_LITERAL = 0, 1
CTQMC_OPT_SCHEDULE, CTQMC_OPT_PANEL_WIDTH, CTQMC_OPT_TIMING, CTQMC_OPT_PATH, CTQMC_OPT_SCRATCH_LIMIT, CTQMC_OPT_ARENA_BYTES, CTQMC_OPT_SPLIT_SLICES = 1, 2, 3, 4, 5, 6, 7
CTQMC_PATH_AUTO, CTQMC_PATH_PANEL, CTQMC_PATH_LARGE, CTQMC_PATH_SMALL, CTQMC_PATH_GROUPED, CTQMC_PATH_SPLIT = 0, 1, 2, 3, 4, 5

CTQMC_CHAIN_OK, CTQMC_CHAIN_BAD_EDIT, CTQMC_CHAIN_NOT_FOUND, CTQMC_CHAIN_LEAF_FULL = 0, 2, 3, 4

EXPORTS = ["ctqmc_load_impurity", "ctqmc_free_impurity", "ctqmc_set_option", "ctqmc_trace_batch", "ctqmc_bound_batch",
           "ctqmc_trace_batch_host", "ctqmc_bound_batch_host", "ctqmc_last_stats", "ctqmc_last_timing", "ctqmc_measure_fp64_peak", "ctqmc_last_error",
           "ctqmc_chains_create", "ctqmc_chains_destroy", "ctqmc_chains_propose", "ctqmc_chains_commit", "ctqmc_chains_trace",
           "ctqmc_chains_stats", "ctqmc_density_size", "ctqmc_density_batch", "ctqmc_density_static_limit", "ctqmc_density_batch_static"]


class CtqmcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ctqmc error {code}: {msg}")
        self.code = code


class _Desc(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("dim", C.c_void_p), ("energy", C.c_void_p), ("n_symbols", C.c_int32),
                ("is_complex", C.c_int32), ("n_blocks", C.c_int64), ("blk_symbol", C.c_void_p), ("blk_src", C.c_void_p),
                ("blk_dst", C.c_void_p), ("blk_offset", C.c_void_p), ("blk_data", C.c_void_p)]


class _Batch(C.Structure):
    _fields_ = [("n_configs", C.c_int64), ("offset", C.c_void_p), ("symbol", C.c_void_p), ("tau", C.c_void_p),
                ("n_ops", C.c_int64), ("max_len", C.c_int32)]


class _ChainsDesc(C.Structure):
    _fields_ = [("n_chains", C.c_int64), ("depth", C.c_int32), ("leaf_capacity", C.c_int32), ("max_edits", C.c_int32),
                ("lazy_rounds", C.c_int32)]


class _EditBatch(C.Structure):
    _fields_ = [("offset", C.c_void_p), ("tau", C.c_void_p), ("symbol", C.c_void_p), ("kind", C.c_void_p), ("n_edits", C.c_int64)]


_lib = None


def library() -> C.CDLL:
    """The loaded shared library; raises if it has not been built (python -m paper_2010_08482_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2010_08482_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        lib.ctqmc_load_impurity.argtypes = [C.POINTER(_Desc), C.c_int, C.POINTER(vp)]
        lib.ctqmc_load_impurity.restype = C.c_int
        lib.ctqmc_free_impurity.argtypes = [vp]
        lib.ctqmc_free_impurity.restype = None
        lib.ctqmc_set_option.argtypes = [vp, C.c_int, i64]
        lib.ctqmc_set_option.restype = C.c_int
        for name in ("ctqmc_trace_batch", "ctqmc_trace_batch_host"):
            fn = getattr(lib, name)
            fn.argtypes = [vp, dbl, C.POINTER(_Batch), vp, vp, vp, vp, vp]
            fn.restype = C.c_int
        for name in ("ctqmc_bound_batch", "ctqmc_bound_batch_host"):
            fn = getattr(lib, name)
            fn.argtypes = [vp, dbl, C.POINTER(_Batch), C.c_int, C.c_int, vp, vp, vp, vp, vp, vp]
            fn.restype = C.c_int
        lib.ctqmc_last_stats.argtypes = [vp, C.POINTER(i64 * 10)]
        lib.ctqmc_last_stats.restype = C.c_int
        lib.ctqmc_last_timing.argtypes = [vp, C.POINTER(dbl * 4)]
        lib.ctqmc_last_timing.restype = C.c_int
        lib.ctqmc_measure_fp64_peak.argtypes = [C.c_int, C.POINTER(dbl), C.POINTER(dbl)]
        lib.ctqmc_measure_fp64_peak.restype = C.c_int
        lib.ctqmc_last_error.argtypes = []
        lib.ctqmc_last_error.restype = C.c_char_p
        lib.ctqmc_chains_create.argtypes = [vp, dbl, C.POINTER(_ChainsDesc), vp, C.POINTER(vp)]
        lib.ctqmc_chains_create.restype = C.c_int
        lib.ctqmc_chains_destroy.argtypes = [vp]
        lib.ctqmc_chains_destroy.restype = None
        lib.ctqmc_chains_propose.argtypes = [vp, C.POINTER(_EditBatch)] + [vp] * 10
        lib.ctqmc_chains_propose.restype = C.c_int
        lib.ctqmc_chains_commit.argtypes = [vp, vp, vp]
        lib.ctqmc_chains_commit.restype = C.c_int
        lib.ctqmc_chains_trace.argtypes = [vp, vp, vp, vp]
        lib.ctqmc_chains_trace.restype = C.c_int
        lib.ctqmc_chains_stats.argtypes = [vp, C.POINTER(i64 * 4)]
        lib.ctqmc_chains_stats.restype = C.c_int
        lib.ctqmc_density_size.argtypes = [vp]
        lib.ctqmc_density_size.restype = i64
        lib.ctqmc_density_batch.argtypes = [vp, dbl, C.POINTER(_Batch), vp, vp, vp, vp, vp, vp]
        lib.ctqmc_density_batch.restype = C.c_int
        lib.ctqmc_density_static_limit.argtypes = []
        lib.ctqmc_density_static_limit.restype = i64
        lib.ctqmc_density_batch_static.argtypes = [vp, dbl, C.POINTER(_Batch), vp, vp, vp, vp, vp, vp]
        lib.ctqmc_density_batch_static.restype = C.c_int
        _lib = lib
    return _lib


def ctqmc_last_error() -> str:
    return library().ctqmc_last_error().decode()


def _check(rc: int):
    if rc != 0:
        raise CtqmcError(rc, ctqmc_last_error())


def _np(a, dtype):
    return np.ascontiguousarray(np.asarray(a), dtype=dtype)


class ImpurityHandle:
    """Owns a `ctqmc_impurity*`.  Created by `ctqmc_load_impurity`."""

    def __init__(self, ptr: int, n_sectors: int, is_complex: bool, device: int):
        self._ptr = C.c_void_p(ptr)
        self.n_sectors = n_sectors
        self.is_complex = is_complex
        self.device = device

    @property
    def ptr(self):
        if not self._ptr:
            raise CtqmcError(CTQMC_ERR_ARG, "impurity handle already freed")
        return self._ptr

    def free(self):
        if self._ptr:
            library().ctqmc_free_impurity(self._ptr)
            self._ptr = C.c_void_p(None)

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def ctqmc_load_impurity(desc, device: int = 0) -> ImpurityHandle:
    """desc: any object with dims, energy, n_symbols, is_complex, blk_symbol, blk_src, blk_dst, blk_offset, blk_data
    (host numpy arrays; e.g. workloads.Impurity).  Copies everything to `device`."""
    dims = _np(desc.dims, np.int32)
    energy = _np(desc.energy, np.float64)
    cplx = bool(desc.is_complex)
    bs, bsrc, bdst = _np(desc.blk_symbol, np.int32), _np(desc.blk_src, np.int32), _np(desc.blk_dst, np.int32)
    boff = _np(desc.blk_offset, np.int64)
    data = _np(desc.blk_data, np.complex128 if cplx else np.float64)
    d = _Desc(len(dims), dims.ctypes.data, energy.ctypes.data, int(desc.n_symbols), int(cplx), len(bs),
              bs.ctypes.data, bsrc.ctypes.data, bdst.ctypes.data, boff.ctypes.data, data.ctypes.data)
    out = C.c_void_p(None)
    _check(library().ctqmc_load_impurity(C.byref(d), int(device), C.byref(out)))
    return ImpurityHandle(out.value, len(dims), cplx, int(device))


def ctqmc_free_impurity(imp: ImpurityHandle):
    imp.free()


def ctqmc_set_option(imp: ImpurityHandle, option: int, value: int):
    _check(library().ctqmc_set_option(imp.ptr, int(option), int(value)))


def ctqmc_last_stats(imp: ImpurityHandle) -> dict:
    buf = (C.c_int64 * 10)()
    _check(library().ctqmc_last_stats(imp.ptr, C.byref(buf)))
    keys = ["strings", "units", "launches", "macs", "alg_flops", "panel_width", "team_warps", "path", "n_exp", "arena_bytes"]
    return dict(zip(keys, [int(x) for x in buf]))


def ctqmc_last_timing(imp: ImpurityHandle) -> dict:
    buf = (C.c_double * 4)()
    _check(library().ctqmc_last_timing(imp.ptr, C.byref(buf)))
    return dict(zip(["route_ms", "chain_ms", "reduce_ms", "total_ms"], [float(x) for x in buf]))


def ctqmc_measure_fp64_peak(device: int = 0) -> dict:
    a, b = C.c_double(0.0), C.c_double(0.0)
    _check(library().ctqmc_measure_fp64_peak(int(device), C.byref(a), C.byref(b)))
    return {"dmma_tflops": a.value, "dfma_tflops": b.value}


def _stream_ptr(stream, host: bool = False):
    if stream is None:
        if host:
            return C.c_void_p(None)   # the legacy default stream
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(stream.cuda_stream))


def _dev_batch(offset, symbol, tau, max_len):
    """n_ops is the length of the symbol tensor (host-known).  max_len: the caller's bound on the longest configuration; a
    caller that does not state it pays one device read here, in the binding (the C call itself never waits for the device)."""
    import torch
    assert offset.is_cuda and offset.dtype == torch.int64 and offset.is_contiguous()
    assert symbol.is_cuda and symbol.dtype == torch.int32 and symbol.is_contiguous()
    assert tau.is_cuda and tau.dtype == torch.float64 and tau.is_contiguous() and tau.numel() == symbol.numel()
    if max_len is None:
        max_len = int((offset[1:] - offset[:-1]).max().item()) if offset.numel() > 1 else 0
        max_len = max(max_len, 1)
    return _Batch(offset.numel() - 1, offset.data_ptr(), symbol.data_ptr(), tau.data_ptr(), symbol.numel(), int(max_len))


def ctqmc_trace_batch(imp: ImpurityHandle, beta: float, offset, symbol, tau, want_survive: bool = True, stream=None,
                      out=None, max_len=None):
    """Device form.  offset int64[B+1], symbol int32[n], tau float64[n]: torch CUDA tensors.  Returns torch CUDA
    tensors (mant[B,2], exp2[B], survive[B,Q] or None, status[B]); asynchronous on `stream` (default: current)."""
    import torch
    B = offset.numel() - 1
    dev = offset.device
    if out is None:
        mant = torch.empty((B, 2), dtype=torch.float64, device=dev)
        exp2 = torch.empty(B, dtype=torch.int64, device=dev)
        surv = torch.empty((B, imp.n_sectors), dtype=torch.uint8, device=dev) if want_survive else None
        status = torch.empty(B, dtype=torch.int32, device=dev)
    else:
        mant, exp2, surv, status = out
    b = _dev_batch(offset, symbol, tau, max_len)
    _check(library().ctqmc_trace_batch(imp.ptr, float(beta), C.byref(b), mant.data_ptr(), exp2.data_ptr(),
                                       surv.data_ptr() if surv is not None else None, status.data_ptr(),
                                       _stream_ptr(stream)))
    return mant, exp2, surv, status


def ctqmc_bound_batch(imp: ImpurityHandle, beta: float, offset, symbol, tau, norm_kind: int = 0, segment_len: int = 1,
                      want_sector: bool = True, stream=None, max_len=None):
    """Device form.  Returns (bound_mant[B], bound_exp2[B], sector_mant[B,Q] | None, sector_exp2[B,Q] | None, status[B])."""
    import torch
    B = offset.numel() - 1
    dev = offset.device
    bm = torch.empty(B, dtype=torch.float64, device=dev)
    be = torch.empty(B, dtype=torch.int64, device=dev)
    sm = torch.empty((B, imp.n_sectors), dtype=torch.float64, device=dev) if want_sector else None
    se = torch.empty((B, imp.n_sectors), dtype=torch.int64, device=dev) if want_sector else None
    status = torch.empty(B, dtype=torch.int32, device=dev)
    b = _dev_batch(offset, symbol, tau, max_len)
    _check(library().ctqmc_bound_batch(imp.ptr, float(beta), C.byref(b), int(norm_kind), int(segment_len),
                                       bm.data_ptr(), be.data_ptr(), sm.data_ptr() if want_sector else None,
                                       se.data_ptr() if want_sector else None, status.data_ptr(), _stream_ptr(stream)))
    return bm, be, sm, se, status


def _host_batch(offset, symbol, tau):
    offset, symbol, tau = _np(offset, np.int64), _np(symbol, np.int32), _np(tau, np.float64)
    keep = (offset, symbol, tau)
    return _Batch(len(offset) - 1, offset.ctypes.data, symbol.ctypes.data if len(symbol) else None,
                  tau.ctypes.data if len(tau) else None, len(symbol), 0), keep


def ctqmc_trace_batch_host(imp: ImpurityHandle, beta: float, offset, symbol, tau, want_survive: bool = True,
                           stream=None, out=None):
    """Host form: numpy in, numpy out; copies and synchronises inside the library.  `out` = (mant, exp2, survive, status)
    numpy arrays to write into (e.g. views of page-locked torch tensors: with page-locked inputs too, the library skips its
    staging copies and overlaps transfers with compute)."""
    b, keep = _host_batch(offset, symbol, tau)
    B = b.n_configs
    if out is not None:
        mant, exp2, surv, status = out
        assert mant.dtype == np.float64 and exp2.dtype == np.int64 and status.dtype == np.int32
        want_survive = surv is not None
    else:
        mant = np.empty((B, 2), np.float64)
        exp2 = np.empty(B, np.int64)
        surv = np.empty((B, imp.n_sectors), np.uint8) if want_survive else None
        status = np.empty(B, np.int32)
    _check(library().ctqmc_trace_batch_host(imp.ptr, float(beta), C.byref(b), mant.ctypes.data, exp2.ctypes.data,
                                            surv.ctypes.data if want_survive else None, status.ctypes.data,
                                            _stream_ptr(stream, host=True)))
    return mant, exp2, surv, status


def ctqmc_bound_batch_host(imp: ImpurityHandle, beta: float, offset, symbol, tau, norm_kind: int = 0,
                           segment_len: int = 1, want_sector: bool = True, stream=None):
    b, keep = _host_batch(offset, symbol, tau)
    B = b.n_configs
    bm = np.empty(B, np.float64)
    be = np.empty(B, np.int64)
    sm = np.empty((B, imp.n_sectors), np.float64) if want_sector else None
    se = np.empty((B, imp.n_sectors), np.int64) if want_sector else None
    status = np.empty(B, np.int32)
    _check(library().ctqmc_bound_batch_host(imp.ptr, float(beta), C.byref(b), int(norm_kind), int(segment_len),
                                            bm.ctypes.data, be.ctypes.data, sm.ctypes.data if want_sector else None,
                                            se.ctypes.data if want_sector else None, status.ctypes.data,
                                            _stream_ptr(stream, host=True)))
    return bm, be, sm, se, status


# ----------------------------------------------------------------------------------------------- chain sets (lazy trace)
class ChainsHandle:
    """Owns a `ctqmc_chains*` (and keeps its impurity alive).  Created by `ctqmc_chains_create`."""

    def __init__(self, ptr: int, imp: ImpurityHandle, n_chains: int):
        self._ptr = C.c_void_p(ptr)
        self.imp = imp
        self.n_chains = n_chains

    @property
    def ptr(self):
        if not self._ptr:
            raise CtqmcError(CTQMC_ERR_ARG, "chain set already destroyed")
        return self._ptr

    def destroy(self):
        if self._ptr:
            library().ctqmc_chains_destroy(self._ptr)
            self._ptr = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def ctqmc_chains_create(imp: ImpurityHandle, beta: float, n_chains: int, depth: int, leaf_capacity: int = 8, max_edits: int = 4,
                        lazy_rounds: int = 1, stream=None) -> ChainsHandle:
    d = _ChainsDesc(int(n_chains), int(depth), int(leaf_capacity), int(max_edits), int(lazy_rounds))
    out = C.c_void_p(None)
    _check(library().ctqmc_chains_create(imp.ptr, float(beta), C.byref(d), _stream_ptr(stream), C.byref(out)))
    return ChainsHandle(out.value, imp, int(n_chains))


def ctqmc_chains_destroy(chains: ChainsHandle):
    chains.destroy()


def ctqmc_chains_propose(chains: ChainsHandle, edit_offset, edit_tau, edit_symbol, edit_kind, log2_threshold=None, stream=None):
    """edit_offset int64[C+1], edit_tau float64[n], edit_symbol int32[n], edit_kind int32[n] (+1 insert, -1 remove),
    log2_threshold float64[C] or None: torch CUDA tensors.  Returns a dict of torch CUDA tensors (accept, decided_by,
    n_sectors_evaluated, bound_mant, bound_exp2, trace_mant[C,2], trace_exp2, status); asynchronous on `stream`."""
    import torch
    nC = chains.n_chains
    dev = edit_offset.device
    assert edit_offset.is_cuda and edit_offset.dtype == torch.int64 and edit_offset.numel() == nC + 1
    assert edit_tau.dtype == torch.float64 and edit_symbol.dtype == torch.int32 and edit_kind.dtype == torch.int32
    assert edit_tau.numel() == edit_symbol.numel() == edit_kind.numel()
    if log2_threshold is not None:
        assert log2_threshold.is_cuda and log2_threshold.dtype == torch.float64 and log2_threshold.numel() == nC
    i32 = dict(dtype=torch.int32, device=dev)
    out = dict(accept=torch.empty(nC, **i32), decided_by=torch.empty(nC, **i32), n_sectors_evaluated=torch.empty(nC, **i32),
               bound_mant=torch.empty(nC, dtype=torch.float64, device=dev), bound_exp2=torch.empty(nC, dtype=torch.int64, device=dev),
               trace_mant=torch.empty((nC, 2), dtype=torch.float64, device=dev), trace_exp2=torch.empty(nC, dtype=torch.int64, device=dev),
               status=torch.empty(nC, **i32))
    n = edit_tau.numel()
    eb = _EditBatch(edit_offset.data_ptr(), edit_tau.data_ptr() if n else None, edit_symbol.data_ptr() if n else None,
                    edit_kind.data_ptr() if n else None, n)
    _check(library().ctqmc_chains_propose(chains.ptr, C.byref(eb), log2_threshold.data_ptr() if log2_threshold is not None else None,
                                          out["accept"].data_ptr(), out["decided_by"].data_ptr(), out["n_sectors_evaluated"].data_ptr(),
                                          out["bound_mant"].data_ptr(), out["bound_exp2"].data_ptr(), out["trace_mant"].data_ptr(),
                                          out["trace_exp2"].data_ptr(), out["status"].data_ptr(), _stream_ptr(stream)))
    return out


def ctqmc_chains_commit(chains: ChainsHandle, mask=None, stream=None):
    """mask: int32[C] torch CUDA tensor, or None = the accept flags of the most recent proposal."""
    import torch
    if mask is not None:
        assert mask.is_cuda and mask.dtype == torch.int32 and mask.numel() == chains.n_chains
    _check(library().ctqmc_chains_commit(chains.ptr, mask.data_ptr() if mask is not None else None, _stream_ptr(stream)))


def ctqmc_chains_trace(chains: ChainsHandle, stream=None):
    import torch
    nC = chains.n_chains
    mant = torch.empty((nC, 2), dtype=torch.float64, device="cuda")
    exp2 = torch.empty(nC, dtype=torch.int64, device="cuda")
    _check(library().ctqmc_chains_trace(chains.ptr, mant.data_ptr(), exp2.data_ptr(), _stream_ptr(stream)))
    return mant, exp2


def ctqmc_chains_stats(chains: ChainsHandle) -> dict:
    buf = (C.c_int64 * 4)()
    _check(library().ctqmc_chains_stats(chains.ptr, C.byref(buf)))
    return dict(zip(["products", "bytes", "launches", "slots_per_chain"], [int(x) for x in buf]))


# ----------------------------------------------------------------------------------------------- reduced density matrix
def ctqmc_density_size(imp: ImpurityHandle) -> int:
    return int(library().ctqmc_density_size(imp.ptr))


def ctqmc_density_batch(imp: ImpurityHandle, beta: float, offset, symbol, tau, w_mant, w_exp2, status, weight=None, rho=None,
                        stream=None, max_len=None):
    """Adds the batch's estimator of the reduced density matrix (Eq. 27) to `rho` (torch CUDA float64 tensor of
    ctqmc_density_size elements, x2 for complex impurities; created zeroed if None) and returns it.  w_mant, w_exp2, status:
    the outputs of ctqmc_trace_batch for the same batch."""
    import torch
    n = ctqmc_density_size(imp) * (2 if imp.is_complex else 1)
    if rho is None:
        rho = torch.zeros(n, dtype=torch.float64, device=offset.device)
    assert rho.is_cuda and rho.dtype == torch.float64 and rho.numel() == n and rho.is_contiguous()
    assert w_mant.dtype == torch.float64 and w_exp2.dtype == torch.int64 and status.dtype == torch.int32
    if weight is not None:
        assert weight.is_cuda and weight.dtype == torch.float64 and weight.numel() == offset.numel() - 1
    b = _dev_batch(offset, symbol, tau, max_len)
    _check(library().ctqmc_density_batch(imp.ptr, float(beta), C.byref(b), w_mant.data_ptr(), w_exp2.data_ptr(), status.data_ptr(),
                                         weight.data_ptr() if weight is not None else None, rho.data_ptr(), _stream_ptr(stream)))
    return rho


def ctqmc_density_static_limit() -> int:
    return int(library().ctqmc_density_static_limit())


def ctqmc_density_batch_static(imp: ImpurityHandle, beta: float, offset, symbol, tau, w_mant, w_exp2, status, rho, weight=None,
                               stream=None, max_len=None):
    """ctqmc_density_batch with its scratch in the library's fixed device array (no cudaMalloc / cudaFree; include/ctqmc.h).
    Nothing is created here either: `rho` is the caller's (zeroed before the first call).  Raises CtqmcError
    (CTQMC_ERR_UNSUPPORTED) when one string's prefix products exceed ctqmc_density_static_limit() bytes."""
    import torch
    n = ctqmc_density_size(imp) * (2 if imp.is_complex else 1)
    assert rho.is_cuda and rho.dtype == torch.float64 and rho.numel() == n and rho.is_contiguous()
    assert w_mant.dtype == torch.float64 and w_exp2.dtype == torch.int64 and status.dtype == torch.int32
    if weight is not None:
        assert weight.is_cuda and weight.dtype == torch.float64 and weight.numel() == offset.numel() - 1
    b = _dev_batch(offset, symbol, tau, max_len)
    _check(library().ctqmc_density_batch_static(imp.ptr, float(beta), C.byref(b), w_mant.data_ptr(), w_exp2.data_ptr(), status.data_ptr(),
                                                weight.data_ptr() if weight is not None else None, rho.data_ptr(), _stream_ptr(stream)))
    return rho
