"""Python binding of libbsramg.so (include/bsr_amg.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; torch is used here for device memory and the
stream only.  There is no CPU fallback: importing works anywhere, but every compute call needs the compiled
library and a CUDA device and raises otherwise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

ERRORS = {1: "NULL", 2: "SHAPE", 3: "BLOCK", 4: "STRUCTURE", 5: "ALLOC", 6: "CUDA", 7: "PLAN", 8: "ALIGN",
          9: "NUMERIC", 10: "LIMIT"}

# every symbol include/bsr_amg.h declares: name -> (restype, argtypes)
_V, _I32, _I64, _D = C.c_void_p, C.c_int32, C.c_int64, C.c_double
_PV, _PI32, _PI64 = C.POINTER(C.c_void_p), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
SYMBOLS = {
    "bsr_last_error": (C.c_char_p, []),
    "bsr_create": (C.c_int, [_PV, _I32, _I32, _I32, _I32, _I64, _V, _V, _V, _V]),
    "bsr_values_changed": (C.c_int, [_V]),
    "bsr_rebind_values": (C.c_int, [_V, _V]),
    "bsr_destroy": (C.c_int, [_V]),
    "bsr_get_info": (C.c_int, [_V, _PI32, _PI32, _PI32, _PI32, _PI64, _PI64]),
    "bsr_spmv": (C.c_int, [_V, _V, _V, _V]),
    "bsr_spmv_t": (C.c_int, [_V, _V, _V, _V]),
    "bsr_transpose_prepare": (C.c_int, [_V, _PI64, _V]),
    "bsr_spmv_host": (C.c_int, [_V, _I32, _V, _V, _V]),
    "bsr_spmv_bytes": (C.c_int64, [_V]),
    "ptap_symbolic": (C.c_int, [_PV, _V, _V, _PI32, _PI64, _V]),
    "ptap_structure": (C.c_int, [_V, _V, _V, _V]),
    "ptap_numeric": (C.c_int, [_V, _V, _V, _V, _V]),
    "ptap_get_info": (C.c_int, [_V, _PI64, _PI64, _PI64, _PI64, _PI64]),
    "ptap_numeric_stage": (C.c_int, [_V, _I32, _V, _V, _V, _V]),
    "ptap_get_ap": (C.c_int, [_V, _V, _V, _V, _V]),
    "ptap_numeric_host": (C.c_int, [_V, _V, _V, _V, _V, _V, _V]),
    "ptap_destroy": (C.c_int, [_V]),
    "ptap_host_plan_build": (C.c_void_p, [_I32, _V, _V, _I32, _V, _V]),
    "ptap_host_plan_get": (C.c_int, [_V, C.c_char_p, _PV, _PI64, _PI32]),
    "ptap_host_stream_stats": (C.c_int, [_V, _I32, _I32, _I32, _I64, _PI64]),
    "ptap_get_schedule": (C.c_int, [_V, _PI64]),
    "bsr_set_option": (C.c_int, [C.c_char_p, _I64]),
    "ptap_host_plan_free": (None, [_V]),
    "vcycle_create": (C.c_int, [_PV, _I32, _PV, _PV, C.POINTER(_D), _I32, _D, _D, _V]),
    "vcycle_refresh": (C.c_int, [_V, _V]),
    "vcycle_status": (C.c_int, [_V, _V]),
    "vcycle_apply": (C.c_int, [_V, _V, _V, _V]),
    "vcycle_smooth": (C.c_int, [_V, _I32, _V, _V, _V]),
    "pcg_solve": (C.c_int, [_V, _V, _V, _I32, _V, _V]),
    "vcycle_apply_host": (C.c_int, [_V, _V, _V, _V]),
    "vcycle_destroy": (C.c_int, [_V]),
    "bsr_set_allocator": (C.c_int, [_V, _V, _V]),
    "bsr_counters": (C.c_int, [_PI64, _PI64]),
    "bsr_measure_fp64_peak": (C.c_int, [C.POINTER(_D), _V]),
    "bsr_measure_fp64_mma_peak": (C.c_int, [C.POINTER(_D), _V]),
    "prolongator_smooth_symbolic": (C.c_int, [_PV, _V, _V, _PI64, _V]),
    "prolongator_smooth_structure": (C.c_int, [_V, _V, _V, _V]),
    "prolongator_smooth_numeric": (C.c_int, [_V, _V, _V, _D, _V, _V]),
    "prolongator_smooth_lambda": (C.c_int, [_V, _V, _V, _I32, C.POINTER(_D), _V]),
    "bsr_lambda_noalloc": (C.c_int, [_V, _V, _I32, _V, _V, _V]),
    "bsr_lambda_noalloc_scratch_doubles": (C.c_int, [_I32, _I32, C.POINTER(_I64)]),
    "prolongator_smooth_status": (C.c_int, [_V, _V]),
    "prolongator_smooth_get_info": (C.c_int, [_V, _PI64, _PI64, _PI32]),
    "prolongator_smooth_destroy": (C.c_int, [_V]),
    "bcoo_plan_create": (C.c_int, [_PV, _I64, _V, _V, _I32, _I32, _I32, _I32, _PI64, _V]),
    "bcoo_structure": (C.c_int, [_V, _V, _V, _V]),
    "bcoo_set_values": (C.c_int, [_V, _V, _V, _V]),
    "bcoo_get_info": (C.c_int, [_V, _PI64, _PI64, _PI64]),
    "bcoo_destroy": (C.c_int, [_V]),
    "bsr_gather_blocks": (C.c_int, [_I64, _V, _I32, _V, _V, _V]),
    "bsr_scatter_add_blocks": (C.c_int, [_I64, _V, _I32, _V, _V, _V]),
    "fem_q1_element_coords": (C.c_int, [_I32, _I32, _I64, _I64, _V, _V, _V]),
    "fem_q1_element_blocks": (C.c_int, [_I32, _I32, _I64, _I64, _V, _V, _I32, _V, _V]),
}


class BsrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libbsramg error {code} ({ERRORS.get(code, '?')}): {msg}")
        self.code = code


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
_workspace = {}      # device pointer -> the torch tensor that backs it (kept alive until the library frees it)
_alloc_cb = _free_cb = None


def _torch_alloc(nbytes, _ctx):
    import torch
    try:
        t = torch.empty(int(nbytes), dtype=torch.uint8, device=torch.device("cuda", torch.cuda.current_device()))
    except Exception:
        return None
    _workspace[t.data_ptr()] = t
    return t.data_ptr()


def _torch_free(ptr, _ctx):
    _workspace.pop(ptr, None)


def use_torch_allocator(enable: bool = True):
    """Library workspace from torch's caching allocator (bsr_set_allocator): "PyTorch for device memory".  On by
    default once a CUDA device is present; `enable=False` goes back to cudaMalloc."""
    global _alloc_cb, _free_cb
    if enable:
        if _alloc_cb is None:
            _alloc_cb, _free_cb = _ALLOC_FN(_torch_alloc), _FREE_FN(_torch_free)
        _check(lib().bsr_set_allocator(C.cast(_alloc_cb, C.c_void_p), C.cast(_free_cb, C.c_void_p), None))
    else:
        _check(lib().bsr_set_allocator(None, None, None))


def _allocator_off_at_exit():
    # blocks still held at interpreter shutdown are left to the process teardown instead of calling back into Python
    try:
        if _lib is not None and _alloc_cb is not None:
            _lib.bsr_set_allocator(None, None, None)
    except Exception:
        pass


import atexit  # noqa: E402
atexit.register(_allocator_off_at_exit)


def workspace_bytes() -> int:
    """Bytes of library workspace currently held through the torch allocator."""
    return sum(int(t.numel()) for t in _workspace.values())


def lib():
    """Loads (building if stale) the CUDA library.  Fails loudly when it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build_cuda()
        L = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)  # AttributeError if the library does not export a declared symbol
            f.restype, f.argtypes = res, args
        _lib = L
        try:
            import torch
            if torch.cuda.is_available():
                use_torch_allocator(True)
        except ImportError:
            pass
    return _lib


def _check(rc: int):
    if rc != 0:
        raise BsrError(rc, lib().bsr_last_error().decode())


def _stream() -> int:
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


def _dev(t):
    """Device pointer of a torch CUDA tensor (None -> null)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def set_option(name: str, value: int):
    """Process-wide option of the cold calls (bsr_set_option): "ptap_force_gather", "ptap_smem_stage1/2"."""
    _check(lib().bsr_set_option(name.encode(), int(value)))


def counters():
    a, b = C.c_int64(), C.c_int64()
    lib().bsr_counters(C.byref(a), C.byref(b))
    return a.value, b.value


NOALLOC_SCRATCH_BYTES = 32 << 20   # BSR_NOALLOC_SCRATCH_BYTES: the fixed work space of bsr_lambda_noalloc


def lambda_noalloc_scratch_bytes(nbrows: int, bs: int) -> int:
    """Work space bsr_lambda_noalloc needs for a matrix of this size (must not exceed NOALLOC_SCRATCH_BYTES)."""
    d = _I64()
    _check(lib().bsr_lambda_noalloc_scratch_doubles(int(nbrows), int(bs), C.byref(d)))
    return d.value * 8


def lambda_noalloc(A: "Bsr", v0, iters: int, out, status=None):
    """Power iteration for lambda of D^-1 A with no allocation anywhere (bsr_lambda_noalloc): `out` is a caller-owned
    DEVICE tensor of one float64, `status` an optional device int32; nothing is synchronised.  Calls that overlap on
    the GPU race on the library's one work array."""
    assert v0.numel() == A.nbrows * A.bs_r and out.numel() >= 1
    _check(lib().bsr_lambda_noalloc(A.h, _dev(v0), int(iters), _dev(out), _dev(status) if status is not None else None,
                                    _stream()))
    return out


def fp64_peak_tflops(mma: bool = False) -> float:
    """Measured fp64 peak of the current device: FMA chains (bsr_measure_fp64_peak) or, mma=True, chains of
    mma.sync m8n8k4 on the fp64 tensor-core path (bsr_measure_fp64_mma_peak)."""
    t = C.c_double()
    fn = lib().bsr_measure_fp64_mma_peak if mma else lib().bsr_measure_fp64_peak
    _check(fn(C.byref(t), _stream()))
    return t.value


class Bsr:
    """A block-CSR matrix on the device (bsr_create).  Keeps the torch tensors it borrows alive."""

    def __init__(self, nbrows, nbcols, bs_r, bs_c, rowptr, colidx, vals):
        import torch
        self.nbrows, self.nbcols, self.bs_r, self.bs_c = int(nbrows), int(nbcols), int(bs_r), int(bs_c)
        self.rowptr, self.colidx, self.vals = rowptr, colidx, vals
        assert rowptr.dtype == torch.int32 and colidx.dtype == torch.int32 and vals.dtype == torch.float64
        self.nnzb = int(colidx.numel())
        h = C.c_void_p()
        _check(lib().bsr_create(C.byref(h), self.nbrows, self.nbcols, self.bs_r, self.bs_c, self.nnzb, _dev(rowptr),
                                _dev(colidx), _dev(vals), _stream()))
        self.h = h

    @classmethod
    def from_host(cls, M, device="cuda"):
        """Upload a host matrix (any object with nbrows, nbcols, bs_r, bs_c, rowptr, colidx, vals numpy arrays)."""
        import torch
        rp = torch.from_numpy(np.ascontiguousarray(M.rowptr, dtype=np.int32)).to(device)
        ci = torch.from_numpy(np.ascontiguousarray(M.colidx, dtype=np.int32)).to(device)
        va = torch.from_numpy(np.ascontiguousarray(M.vals, dtype=np.float64).reshape(-1)).to(device)
        return cls(M.nbrows, M.nbcols, M.bs_r, M.bs_c, rp, ci, va)

    def close(self):
        if getattr(self, "h", None):
            lib().bsr_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def values_changed(self):
        _check(lib().bsr_values_changed(self.h))

    def rebind_values(self, vals):
        """The values now live in another device tensor of the same size (bsr_rebind_values); bumps the state."""
        assert vals.numel() == self.vals.numel() and vals.dtype == self.vals.dtype and vals.is_cuda
        _check(lib().bsr_rebind_values(self.h, _dev(vals)))
        self.vals = vals

    def set_values(self, host_vals):
        """Rewrite the values in place from a host array and bump the state counter."""
        import torch
        self.vals.copy_(torch.from_numpy(np.ascontiguousarray(host_vals, dtype=np.float64).reshape(-1)))
        self.values_changed()

    @property
    def state(self) -> int:
        s = C.c_int64()
        _check(lib().bsr_get_info(self.h, None, None, None, None, None, C.byref(s)))
        return s.value

    def spmv_bytes(self) -> int:
        return int(lib().bsr_spmv_bytes(self.h))

    def spmv(self, x, y=None):
        """y = A x (bsr_spmv)."""
        import torch
        if y is None:
            y = torch.empty(self.nbrows * self.bs_r, dtype=torch.float64, device=x.device)
        assert x.numel() == self.nbcols * self.bs_c and y.numel() == self.nbrows * self.bs_r
        _check(lib().bsr_spmv(self.h, _dev(x), _dev(y), _stream()))
        return y

    def spmv_t(self, x, y=None):
        """y = A^T x on the cached explicit transpose (bsr_spmv_t)."""
        import torch
        if y is None:
            y = torch.empty(self.nbcols * self.bs_c, dtype=torch.float64, device=x.device)
        assert x.numel() == self.nbrows * self.bs_r and y.numel() == self.nbcols * self.bs_c
        _check(lib().bsr_spmv_t(self.h, _dev(x), _dev(y), _stream()))
        return y

    def transpose_prepare(self) -> int:
        n = C.c_int64()
        _check(lib().bsr_transpose_prepare(self.h, C.byref(n), _stream()))
        return n.value

    def spmv_host(self, h_x: np.ndarray, h_y: np.ndarray, trans: bool = False):
        """End to end with host vectors (bsr_spmv_host)."""
        assert h_x.dtype == np.float64 and h_y.dtype == np.float64
        _check(lib().bsr_spmv_host(self.h, 1 if trans else 0, h_x.ctypes.data, h_y.ctypes.data, _stream()))
        return h_y


class PtapPlan:
    """Cached symbolic structure and block coordinate plan of A_c = P^T A P (ptap_symbolic)."""

    def __init__(self, A: Bsr, P: Bsr):
        import torch
        self.A, self.P = A, P
        h, nbr, nnz = C.c_void_p(), C.c_int32(), C.c_int64()
        _check(lib().ptap_symbolic(C.byref(h), A.h, P.h, C.byref(nbr), C.byref(nnz), _stream()))
        self.h = h
        self.nbrows_c, self.nnzb_c, self.bs_c = nbr.value, nnz.value, P.bs_c
        dev = A.vals.device
        self.rowptr_c = torch.empty(self.nbrows_c + 1, dtype=torch.int32, device=dev)
        self.colidx_c = torch.empty(self.nnzb_c, dtype=torch.int32, device=dev)
        _check(lib().ptap_structure(self.h, _dev(self.rowptr_c), _dev(self.colidx_c), _stream()))

    def close(self):
        if getattr(self, "h", None):
            lib().ptap_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        v = [C.c_int64() for _ in range(5)]
        _check(lib().ptap_get_info(self.h, *[C.byref(t) for t in v]))
        return dict(nnzb_ap=v[0].value, n_products_1=v[1].value, n_products_2=v[2].value,
                    algorithmic_bytes=v[3].value, n_r_value_builds=v[4].value)

    def schedule(self) -> dict:
        o = (C.c_int64 * 8)()
        _check(lib().ptap_get_schedule(self.h, o))
        k = ["staged", "bricks", "reserved", "smem"]
        return {1: dict(zip(k, [int(v) for v in o[:4]])), 2: dict(zip(k, [int(v) for v in o[4:]]))}

    def new_values(self):
        import torch
        return torch.empty(self.nnzb_c * self.bs_c * self.bs_c, dtype=torch.float64, device=self.A.vals.device)

    def numeric(self, vals_c=None):
        """vals_c = values of P^T A P for the current values of A and P (ptap_numeric)."""
        if vals_c is None:
            vals_c = self.new_values()
        _check(lib().ptap_numeric(self.h, self.A.h, self.P.h, _dev(vals_c), _stream()))
        return vals_c

    def numeric_stage(self, stage: int, vals_c=None):
        _check(lib().ptap_numeric_stage(self.h, stage, self.A.h, self.P.h, _dev(vals_c), _stream()))

    def numeric_host(self, h_vals_a: np.ndarray, h_vals_c: np.ndarray, vals_c):
        _check(lib().ptap_numeric_host(self.h, self.A.h, self.P.h, h_vals_a.ctypes.data, h_vals_c.ctypes.data,
                                       _dev(vals_c), _stream()))
        return h_vals_c

    def coarse_matrix(self, vals_c) -> Bsr:
        """Wrap A_c (structure of the plan, given values) as a Bsr."""
        return Bsr(self.nbrows_c, self.nbrows_c, self.bs_c, self.bs_c, self.rowptr_c, self.colidx_c, vals_c)

    def ap_host(self):
        """(rowptr, colidx, vals) of the cached AP copied to the host (tests)."""
        import torch
        n, bf, bc = self.info()["nnzb_ap"], self.A.bs_r, self.P.bs_c
        dev = self.A.vals.device
        rp = torch.empty(self.A.nbrows + 1, dtype=torch.int32, device=dev)
        ci = torch.empty(n, dtype=torch.int32, device=dev)
        va = torch.empty(n * bf * bc, dtype=torch.float64, device=dev)
        _check(lib().ptap_get_ap(self.h, _dev(rp), _dev(ci), _dev(va), _stream()))
        return rp.cpu().numpy(), ci.cpu().numpy(), va.cpu().numpy().reshape(n, bf, bc)


class ProlongatorSmoother:
    """P = (I - omega D^-1 A) P~ on the device (prolongator_smooth_*)."""

    def __init__(self, A: Bsr, P_tent: Bsr):
        import torch
        self.A, self.Pt = A, P_tent
        h, nnz = C.c_void_p(), C.c_int64()
        _check(lib().prolongator_smooth_symbolic(C.byref(h), A.h, P_tent.h, C.byref(nnz), _stream()))
        self.h, self.nnzb_p = h, nnz.value
        dev = A.vals.device
        self.rowptr_p = torch.empty(A.nbrows + 1, dtype=torch.int32, device=dev)
        self.colidx_p = torch.empty(self.nnzb_p, dtype=torch.int32, device=dev)
        _check(lib().prolongator_smooth_structure(self.h, _dev(self.rowptr_p), _dev(self.colidx_p), _stream()))

    def close(self):
        if getattr(self, "h", None):
            lib().prolongator_smooth_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        a, b, c = C.c_int64(), C.c_int64(), C.c_int32()
        _check(lib().prolongator_smooth_get_info(self.h, C.byref(a), C.byref(b), C.byref(c)))
        return dict(n_products=a.value, algorithmic_bytes=b.value, staged=bool(c.value))

    def new_values(self):
        import torch
        return torch.empty(self.nnzb_p * self.Pt.bs_r * self.Pt.bs_c, dtype=torch.float64, device=self.A.vals.device)

    def numeric(self, omega: float, vals_p=None, check: bool = False):
        """vals_p = values of the smoothed prolongator for the current A, P~ (prolongator_smooth_numeric)."""
        if vals_p is None:
            vals_p = self.new_values()
        _check(lib().prolongator_smooth_numeric(self.h, self.A.h, self.Pt.h, float(omega), _dev(vals_p), _stream()))
        if check:
            _check(lib().prolongator_smooth_status(self.h, _stream()))
        return vals_p

    def lambda_estimate(self, v0, iters: int = 20) -> float:
        """lambda of D^-1 A after `iters` power iterations from v0 on the device (prolongator_smooth_lambda);
        omega = 4 / (3 lambda)."""
        lam = C.c_double()
        assert v0.numel() == self.A.nbrows * self.A.bs_r
        _check(lib().prolongator_smooth_lambda(self.h, self.A.h, _dev(v0), int(iters), C.byref(lam), _stream()))
        return lam.value

    def matrix(self, vals_p) -> Bsr:
        """Wrap P (structure of the plan, given values) as a Bsr."""
        return Bsr(self.A.nbrows, self.Pt.nbcols, self.Pt.bs_r, self.Pt.bs_c, self.rowptr_p, self.colidx_p, vals_p)


class BcooPlan:
    """Blocked COO assembly plan (bcoo_plan_create): coordinates declared once."""

    def __init__(self, brow, bcol, nbrows: int, nbcols: int, bs_r: int, bs_c: int):
        import torch
        assert brow.dtype == torch.int32 and bcol.dtype == torch.int32 and brow.numel() == bcol.numel()
        self.nbrows, self.nbcols, self.bs_r, self.bs_c, self.n = nbrows, nbcols, bs_r, bs_c, int(brow.numel())
        h, nnz = C.c_void_p(), C.c_int64()
        _check(lib().bcoo_plan_create(C.byref(h), self.n, _dev(brow), _dev(bcol), nbrows, nbcols, bs_r, bs_c,
                                      C.byref(nnz), _stream()))
        self.h, self.nnzb = h, nnz.value
        self.rowptr = torch.empty(nbrows + 1, dtype=torch.int32, device=brow.device)
        self.colidx = torch.empty(self.nnzb, dtype=torch.int32, device=brow.device)
        _check(lib().bcoo_structure(self.h, _dev(self.rowptr), _dev(self.colidx), _stream()))

    def close(self):
        if getattr(self, "h", None):
            lib().bcoo_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        v = [C.c_int64() for _ in range(3)]
        _check(lib().bcoo_get_info(self.h, *[C.byref(t) for t in v]))
        return dict(n_contrib=v[0].value, nnzb=v[1].value, algorithmic_bytes=v[2].value)

    def new_values(self):
        import torch
        return torch.empty(self.nnzb * self.bs_r * self.bs_c, dtype=torch.float64, device=self.rowptr.device)

    def set_values(self, stream, vals=None):
        """vals = the assembled block values for this stream of contribution blocks (bcoo_set_values)."""
        assert stream.numel() == self.n * self.bs_r * self.bs_c
        if vals is None:
            vals = self.new_values()
        _check(lib().bcoo_set_values(self.h, _dev(stream), _dev(vals), _stream()))
        return vals

    def matrix(self, vals) -> Bsr:
        return Bsr(self.nbrows, self.nbcols, self.bs_r, self.bs_c, self.rowptr, self.colidx, vals)


def gather_blocks(idx, bs: int, src, dst=None):
    """dst block t = src block idx[t] (bsr_gather_blocks): device-side packing for the halo / P_oth exchange."""
    import torch
    n = int(idx.numel())
    if dst is None:
        dst = torch.empty(n * bs, dtype=torch.float64, device=src.device)
    assert idx.dtype == torch.int32 and dst.numel() == n * bs
    _check(lib().bsr_gather_blocks(n, _dev(idx), bs, _dev(src), _dev(dst), _stream()))
    return dst


def scatter_add_blocks(idx, bs: int, src, dst):
    """dst block idx[t] += src block t, idx distinct (bsr_scatter_add_blocks): the owner's side of the reduce."""
    import torch
    n = int(idx.numel())
    assert idx.dtype == torch.int32 and src.numel() == n * bs
    _check(lib().bsr_scatter_add_blocks(n, _dev(idx), bs, _dev(src), _dev(dst), _stream()))
    return dst


def fem_q1_coords(d: int, ne: int, e0: int, e1: int, device="cuda"):
    """(brow, bcol) of the Q1 element contributions of elements [e0, e1) (fem_q1_element_coords)."""
    import torch
    n = (e1 - e0) * 4 ** d
    brow = torch.empty(n, dtype=torch.int32, device=device)
    bcol = torch.empty(n, dtype=torch.int32, device=device)
    _check(lib().fem_q1_element_coords(d, ne, e0, e1, _dev(brow), _dev(bcol), _stream()))
    return brow, bcol


def fem_q1_blocks(d: int, ne: int, e0: int, e1: int, Ke, E, dirichlet: bool, out=None):
    """The stream of E_e * Ke[a][b] blocks of elements [e0, e1) (fem_q1_element_blocks); Ke, E device tensors."""
    import torch
    n = (e1 - e0) * 4 ** d * d * d
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=Ke.device)
    assert out.numel() == n
    _check(lib().fem_q1_element_blocks(d, ne, e0, e1, _dev(Ke), _dev(E), 1 if dirichlet else 0, _dev(out), _stream()))
    return out


class HostPlan:
    """The host (integer) part of ptap_symbolic on host arrays -- usable without a GPU (tests of the plan)."""
    NAMES = ["rowptr_ap", "colidx_ap", "rowidx_ap", "rowptr_c", "colidx_c", "rowidx_c", "rowptr_r", "colidx_r",
             "perm_r", "pairptr1", "k1", "q1", "pstart", "pairptr2", "t2", "s2", "apstart"]

    def __init__(self, A, P):
        ra, ca = np.ascontiguousarray(A.rowptr, np.int32), np.ascontiguousarray(A.colidx, np.int32)
        rp, cp = np.ascontiguousarray(P.rowptr, np.int32), np.ascontiguousarray(P.colidx, np.int32)
        h = lib().ptap_host_plan_build(A.nbrows, ra.ctypes.data, ca.ctypes.data, P.nbcols, rp.ctypes.data,
                                       cp.ctypes.data)
        if not h:
            raise BsrError(-1, lib().bsr_last_error().decode())
        try:
            for name in self.NAMES:
                ptr, cnt, eb = C.c_void_p(), C.c_int64(), C.c_int32()
                _check(lib().ptap_host_plan_get(h, name.encode(), C.byref(ptr), C.byref(cnt), C.byref(eb)))
                dt = np.int32 if eb.value == 4 else np.uint16
                if cnt.value:
                    buf = (C.c_char * (cnt.value * eb.value)).from_address(ptr.value)
                    arr = np.frombuffer(buf, dtype=dt).copy()
                else:
                    arr = np.empty(0, dt)
                setattr(self, name, arr)
            self.stream_stats = {}
            if getattr(A, "bs_r", None) and getattr(P, "bs_c", None):
                for stage, budget in ((1, 112 * 1024), (2, 75000)):
                    o = (C.c_int64 * 8)()
                    _check(lib().ptap_host_stream_stats(h, A.bs_r, P.bs_c, stage, budget, o))
                    self.stream_stats[stage] = dict(zip(["ok", "bricks", "chunks", "max_smem", "mask_bits", "lanes",
                                                         "passes", "steps"], [int(v) for v in o]))
        finally:
            lib().ptap_host_plan_free(h)


class VCycle:
    """V-cycle preconditioner over a hierarchy of Bsr operators and prolongators (vcycle_create)."""

    def __init__(self, As, Ps, lambdas, cheb_degree: int = 2, lo: float = 0.1, hi: float = 1.1):
        assert len(Ps) == len(As) - 1 and len(lambdas) >= len(Ps)
        self.As, self.Ps = list(As), list(Ps)
        n = len(As)
        a = (C.c_void_p * n)(*[A.h for A in As])
        p = (C.c_void_p * max(n - 1, 1))(*[P.h for P in Ps])
        lam = (C.c_double * max(n - 1, 1))(*[float(v) for v in lambdas[:n - 1]])
        h = C.c_void_p()
        _check(lib().vcycle_create(C.byref(h), n, a, p, lam, cheb_degree, lo, hi, _stream()))
        self.h = h
        self.n = As[0].nbrows * As[0].bs_r

    def close(self):
        if getattr(self, "h", None):
            lib().vcycle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def refresh(self, check: bool = True):
        _check(lib().vcycle_refresh(self.h, _stream()))
        if check:
            _check(lib().vcycle_status(self.h, _stream()))

    def apply(self, b, x=None):
        """x = M^-1 b, one V-cycle from a zero guess (vcycle_apply)."""
        import torch
        if x is None:
            x = torch.empty_like(b)
        assert b.numel() == self.n and x.numel() == self.n
        _check(lib().vcycle_apply(self.h, _dev(b), _dev(x), _stream()))
        return x

    def smooth(self, level: int, b, x):
        _check(lib().vcycle_smooth(self.h, level, _dev(b), _dev(x), _stream()))
        return x

    def pcg(self, b, iters: int = 20):
        """(x, residual history) of `iters` PCG iterations with the V-cycle as preconditioner (pcg_solve)."""
        import torch
        x = torch.empty_like(b)
        hist = torch.empty(iters + 1, dtype=torch.float64, device=b.device)
        _check(lib().pcg_solve(self.h, _dev(b), _dev(x), iters, _dev(hist), _stream()))
        return x, hist

    def apply_host(self, h_b: np.ndarray, h_x: np.ndarray):
        _check(lib().vcycle_apply_host(self.h, h_b.ctypes.data, h_x.ctypes.data, _stream()))
        return h_x
