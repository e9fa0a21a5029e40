"""ctypes binding of the CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares nothing with the CUDA path and imports nothing from paper_2606_24748_b200; matrices come in as any
object with the attributes nbrows, nbcols, bs_r, bs_c, rowptr, colidx, vals (numpy arrays).
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(SRC) > os.path.getmtime(LIB):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-o", LIB, SRC]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("oracle build failed")
    return LIB


class _Bsr(C.Structure):
    _fields_ = [("nbrows", C.c_int32), ("nbcols", C.c_int32), ("bs_r", C.c_int32), ("bs_c", C.c_int32),
                ("nnzb", C.c_int64), ("rowptr", C.c_void_p), ("colidx", C.c_void_p), ("vals", C.c_void_p)]


@dataclasses.dataclass
class OBsr:
    nbrows: int
    nbcols: int
    bs_r: int
    bs_c: int
    rowptr: np.ndarray
    colidx: np.ndarray
    vals: np.ndarray  # (nnzb, bs_r, bs_c)

    @property
    def nnzb(self) -> int:
        return int(self.colidx.shape[0])


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        P = C.POINTER(_Bsr)
        V = C.c_void_p
        lib.orc_set_threads.argtypes = [C.c_int]
        lib.orc_spmv.argtypes = [P, V, V]
        lib.orc_spmv_t.argtypes = [P, V, V]
        lib.orc_spmv_fast.argtypes = [P, V, V]
        lib.orc_transpose.argtypes = [P, V, V, V]
        lib.orc_spgemm_symbolic.restype = C.c_int64
        lib.orc_spgemm_symbolic.argtypes = [C.c_int32, V, V, V, V, V, V]
        lib.orc_ptap_form1.argtypes = [P, P, V, V, V, C.c_int32, V]
        lib.orc_ptap_form2.argtypes = [P, P, P, V, V, V, V, V, V]
        lib.orc_power_lambda.restype = C.c_double
        lib.orc_power_lambda.argtypes = [P, V, C.c_int]
        lib.orc_prolongator_smooth.argtypes = [P, P, C.c_double, V, V, V]
        lib.orc_bcoo_structure.restype = C.c_int64
        lib.orc_bcoo_structure.argtypes = [C.c_int64, V, V, C.c_int32, C.c_int32, V, V]
        lib.orc_bcoo_sum.argtypes = [C.c_int64, V, V, V, C.c_int32, C.c_int32, C.c_int32, V, V, V]
        lib.orc_hier_create.restype = C.c_void_p
        lib.orc_hier_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double]
        lib.orc_hier_destroy.argtypes = [V]
        lib.orc_hier_set_level.argtypes = [V, C.c_int, P, P, C.c_double]
        lib.orc_hier_setup.argtypes = [V]
        lib.orc_smooth.argtypes = [V, C.c_int, V, V]
        lib.orc_vcycle.argtypes = [V, V, V]
        lib.orc_pcg.argtypes = [V, V, V, C.c_int, V]
        _lib = lib
    return _lib


class _Held:
    """A C view of a matrix plus the contiguous arrays that back it."""

    def __init__(self, M):
        self.rowptr = np.ascontiguousarray(M.rowptr, dtype=np.int32)
        self.colidx = np.ascontiguousarray(M.colidx, dtype=np.int32)
        self.vals = np.ascontiguousarray(M.vals, dtype=np.float64)
        self.c = _Bsr(M.nbrows, M.nbcols, M.bs_r, M.bs_c, int(self.colidx.shape[0]), self.rowptr.ctypes.data,
                      self.colidx.ctypes.data, self.vals.ctypes.data)


def _vec(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


def set_threads(n: int = 0) -> int:
    """OpenMP threads of the row-parallel routines from now on (0: default); returns the count in effect."""
    return int(_load().orc_set_threads(int(n)))


def spmv(A, x) -> np.ndarray:
    """y = A x."""
    h, x = _Held(A), _vec(x)
    assert x.shape[0] == A.nbcols * A.bs_c
    y = np.empty(A.nbrows * A.bs_r)
    _load().orc_spmv(h.c, x.ctypes.data, y.ctypes.data)
    return y


def spmv_t(A, x) -> np.ndarray:
    """y = A^T x (restriction)."""
    h, x = _Held(A), _vec(x)
    assert x.shape[0] == A.nbrows * A.bs_r
    y = np.empty(A.nbcols * A.bs_c)
    _load().orc_spmv_t(h.c, x.ctypes.data, y.ctypes.data)
    return y


def spmv_fast(A, x, y=None, held=None) -> np.ndarray:
    """Same definition with double accumulators, row-parallel: the timed CPU baseline."""
    h = held or _Held(A)
    x = _vec(x)
    if y is None:
        y = np.empty(A.nbrows * A.bs_r)
    _load().orc_spmv_fast(h.c, x.ctypes.data, y.ctypes.data)
    return y


def transpose(A, structure_only: bool = False) -> OBsr:
    """Explicit R = A^T with sorted rows."""
    h = _Held(A)
    rp = np.empty(A.nbcols + 1, dtype=np.int32)
    ci = np.empty(h.c.nnzb, dtype=np.int32)
    va = np.empty((h.c.nnzb, A.bs_c, A.bs_r))
    _load().orc_transpose(h.c, rp.ctypes.data, ci.ctypes.data, None if structure_only else va.ctypes.data)
    return OBsr(A.nbcols, A.nbrows, A.bs_c, A.bs_r, rp, ci, va)


def spgemm_symbolic(nrows_a, rowptr_a, colidx_a, rowptr_b, colidx_b):
    """Boolean pattern of A*B with ascending columns -> (rowptr, colidx)."""
    ra, ca = np.ascontiguousarray(rowptr_a, np.int32), np.ascontiguousarray(colidx_a, np.int32)
    rb, cb = np.ascontiguousarray(rowptr_b, np.int32), np.ascontiguousarray(colidx_b, np.int32)
    rc = np.empty(nrows_a + 1, dtype=np.int32)
    n = _load().orc_spgemm_symbolic(nrows_a, ra.ctypes.data, ca.ctypes.data, rb.ctypes.data, cb.ctypes.data,
                                    rc.ctypes.data, None)
    cc = np.empty(n, dtype=np.int32)
    _load().orc_spgemm_symbolic(nrows_a, ra.ctypes.data, ca.ctypes.data, rb.ctypes.data, cb.ctypes.data,
                                rc.ctypes.data, cc.ctypes.data)
    return rc, cc


def ptap_symbolic(A, P):
    """Structures of AP = A*P and A_c = P^T*(AP): ((rowptr_ap, colidx_ap), (rowptr_c, colidx_c))."""
    R = transpose(P, structure_only=True)
    ap = spgemm_symbolic(A.nbrows, A.rowptr, A.colidx, P.rowptr, P.colidx)
    ac = spgemm_symbolic(R.nbrows, R.rowptr, R.colidx, ap[0], ap[1])
    return ap, ac


def ptap(A, P, structure=None, rows=None) -> OBsr:
    """A_c = P^T A P, form 1 (long double, serial).  rows: optional list of coarse rows to compute (others 0)."""
    if structure is None:
        structure = ptap_symbolic(A, P)[1]
    rc, cc = structure
    ha, hp = _Held(A), _Held(P)
    vals = np.zeros((cc.shape[0], P.bs_c, P.bs_c))
    if rows is None:
        nsel, sel = -1, None
    else:
        selarr = np.ascontiguousarray(rows, dtype=np.int32)
        nsel, sel = int(selarr.shape[0]), selarr.ctypes.data
    rcode = _load().orc_ptap_form1(ha.c, hp.c, rc.ctypes.data, cc.ctypes.data, vals.ctypes.data, nsel, sel)
    if rcode != 0:
        raise RuntimeError(f"orc_ptap_form1 failed ({rcode})")
    return OBsr(P.nbcols, P.nbcols, P.bs_c, P.bs_c, rc, cc, vals)


class PtapForm2:
    """Form 2 with everything symbolic prepared once; run() is the timed CPU baseline (double, OpenMP)."""

    def __init__(self, A, P):
        self.A, self.P = A, P
        self.R = transpose(P)
        (self.rap, self.cap), (self.rc, self.cc) = ptap_symbolic(A, P)
        self.vals_ap = np.empty((self.cap.shape[0], A.bs_r, P.bs_c))
        self.vals_c = np.empty((self.cc.shape[0], P.bs_c, P.bs_c))
        self.ha, self.hp, self.hr = _Held(A), _Held(P), _Held(self.R)

    def run(self, A_vals=None) -> OBsr:
        if A_vals is not None:
            self.ha.vals = np.ascontiguousarray(A_vals, dtype=np.float64)
            self.ha.c.vals = self.ha.vals.ctypes.data
        rcode = _load().orc_ptap_form2(self.ha.c, self.hp.c, self.hr.c, self.rap.ctypes.data, self.cap.ctypes.data,
                                       self.vals_ap.ctypes.data, self.rc.ctypes.data, self.cc.ctypes.data,
                                       self.vals_c.ctypes.data)
        if rcode != 0:
            raise RuntimeError(f"orc_ptap_form2 failed ({rcode})")
        return OBsr(self.P.nbcols, self.P.nbcols, self.P.bs_c, self.P.bs_c, self.rc, self.cc, self.vals_c)


def power_lambda(A, v0, iters: int = 20) -> float:
    """lambda of D^-1 A after `iters` power iterations from v0 (reading R10); omega = 4 / (3 lambda)."""
    h, v0 = _Held(A), _vec(v0)
    assert v0.shape[0] == A.nbrows * A.bs_r
    lam = float(_load().orc_power_lambda(h.c, v0.ctypes.data, int(iters)))
    if lam < 0:
        raise RuntimeError(f"orc_power_lambda failed ({lam})")
    return lam


def prolongator_smooth(A, Pt, omega: float) -> OBsr:
    """P = (I - omega D^-1 A) P~ on the boolean pattern of A*P~ (D the block diagonal, R11)."""
    rp, cp = spgemm_symbolic(A.nbrows, A.rowptr, A.colidx, Pt.rowptr, Pt.colidx)
    ha, ht = _Held(A), _Held(Pt)
    vals = np.zeros((cp.shape[0], Pt.bs_r, Pt.bs_c))
    rcode = _load().orc_prolongator_smooth(ha.c, ht.c, float(omega), rp.ctypes.data, cp.ctypes.data, vals.ctypes.data)
    if rcode != 0:
        raise RuntimeError(f"orc_prolongator_smooth failed ({rcode})")
    return OBsr(Pt.nbrows, Pt.nbcols, Pt.bs_r, Pt.bs_c, rp, cp, vals)


def bcoo_assemble(brow, bcol, stream, nbrows: int, nbcols: int, structure=None) -> OBsr:
    """Blocked COO assembly: one block per distinct (brow, bcol), each the sum of the
    stream blocks (n, bs_r, bs_c) that carry its coordinate."""
    brow, bcol = np.ascontiguousarray(brow, np.int32), np.ascontiguousarray(bcol, np.int32)
    stream = np.ascontiguousarray(stream, np.float64)
    n, bs_r, bs_c = stream.shape
    assert brow.shape[0] == n and bcol.shape[0] == n
    lib = _load()
    if structure is None:
        rp = np.empty(nbrows + 1, dtype=np.int32)
        nnzb = lib.orc_bcoo_structure(n, brow.ctypes.data, bcol.ctypes.data, nbrows, nbcols, rp.ctypes.data, None)
        if nnzb < 0:
            raise RuntimeError("orc_bcoo_structure: coordinate out of range")
        ci = np.empty(nnzb, dtype=np.int32)
        lib.orc_bcoo_structure(n, brow.ctypes.data, bcol.ctypes.data, nbrows, nbcols, rp.ctypes.data, ci.ctypes.data)
    else:
        rp, ci = (np.ascontiguousarray(t, np.int32) for t in structure)
    vals = np.empty((ci.shape[0], bs_r, bs_c))
    rcode = lib.orc_bcoo_sum(n, brow.ctypes.data, bcol.ctypes.data, stream.ctypes.data, bs_r, bs_c, nbrows,
                             rp.ctypes.data, ci.ctypes.data, vals.ctypes.data)
    if rcode != 0:
        raise RuntimeError(f"orc_bcoo_sum failed ({rcode})")
    return OBsr(nbrows, nbcols, bs_r, bs_c, rp, ci, vals)


class Hierarchy:
    """Block-Jacobi/Chebyshev V-cycle and PCG over levels A_0..A_{L-1} with prolongators P_0..P_{L-2}."""

    def __init__(self, As, Ps, lambdas, cheb_degree: int = 2, lo: float = 0.1, hi: float = 1.1):
        assert len(Ps) == len(As) - 1 and len(lambdas) >= len(As) - 1
        self._lib = _load()
        self._held = []
        self.n = As[0].nbrows * As[0].bs_r
        self._h = self._lib.orc_hier_create(len(As), cheb_degree, lo, hi)
        for l, A in enumerate(As):
            ha = _Held(A)
            hp = _Held(Ps[l]) if l < len(Ps) else None
            self._held += [ha, hp]
            lam = lambdas[l] if l < len(lambdas) else 0.0
            self._lib.orc_hier_set_level(self._h, l, ha.c, hp.c if hp else None, lam)
        self.setup()

    def setup(self):
        rc = self._lib.orc_hier_setup(self._h)
        if rc != 0:
            raise RuntimeError(f"orc_hier_setup failed ({rc})")

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.orc_hier_destroy(self._h)
            self._h = None

    def smooth(self, level: int, b, x) -> np.ndarray:
        b, x = _vec(b), _vec(x).copy()
        self._lib.orc_smooth(self._h, level, b.ctypes.data, x.ctypes.data)
        return x

    def vcycle(self, b) -> np.ndarray:
        b = _vec(b)
        x = np.empty(self.n)
        self._lib.orc_vcycle(self._h, b.ctypes.data, x.ctypes.data)
        return x

    def pcg(self, b, iters: int = 20):
        b = _vec(b)
        x = np.empty(self.n)
        hist = np.empty(iters + 1)
        self._lib.orc_pcg(self._h, b.ctypes.data, x.ctypes.data, iters, hist.ctypes.data)
        return x, hist
