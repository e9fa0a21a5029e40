"""Seeded synthetic inputs: the five BASELINE.json configs as host (numpy) BSR matrices and vectors.

Thin ctypes binding over gen/libelastgen.so (gen/elasticity_gen.cpp).  This module makes INPUTS only; it
holds none of the hot path and is the one piece shared by the tests (oracle side and CUDA side) and bench.py.
The paper measures on PETSc's ex56 elasticity programs; these procedurally generated Q1
elasticity problems stand in for them ("Input recipe").
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        path = _build.build_gen()
        lib = C.CDLL(path)
        lib.egen_create2.restype = C.c_void_p
        lib.egen_create2.argtypes = [C.c_int, C.c_int, C.c_double, C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int]
        lib.egen_destroy.argtypes = [C.c_void_p]
        lib.egen_error.restype = C.c_char_p
        lib.egen_error.argtypes = [C.c_void_p]
        lib.egen_nlevels.argtypes = [C.c_void_p]
        lib.egen_matrix.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.POINTER(C.c_int32)] * 4 + [
            C.POINTER(C.c_int64), C.POINTER(C.POINTER(C.c_int32)), C.POINTER(C.POINTER(C.c_int32)),
            C.POINTER(C.POINTER(C.c_double))]
        lib.egen_set_operator.argtypes = [C.c_void_p, C.c_int, C.c_int32, C.c_int32, C.c_int64, C.c_void_p,
                                          C.c_void_p, C.c_void_p]
        lib.egen_build_prolongator.argtypes = [C.c_void_p, C.c_int]
        lib.egen_level_info.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                        C.POINTER(C.c_int32), C.POINTER(C.c_int32 * 3), C.POINTER(C.c_double),
                                        C.POINTER(C.c_double)]
        lib.egen_level_arrays.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.POINTER(C.c_double)),
                                          C.POINTER(C.POINTER(C.c_double)), C.POINTER(C.POINTER(C.c_int32))]
        lib.egen_element_matrix2.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_void_p]
        lib.egen_element_stream.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.egen_element_data.argtypes = [C.c_void_p, C.POINTER(C.POINTER(C.c_double)),
                                          C.POINTER(C.POINTER(C.c_double))]
        lib.egen_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_double, C.c_double, C.c_void_p]
        _lib = lib
    return _lib


@dataclasses.dataclass
class HostBSR:
    """Block-CSR on the host: int32 rowptr/colidx, fp64 row-major blocks."""
    nbrows: int
    nbcols: int
    bs_r: int
    bs_c: int
    rowptr: np.ndarray
    colidx: np.ndarray
    vals: np.ndarray  # shape (nnzb, bs_r, bs_c)

    @property
    def nnzb(self) -> int:
        return int(self.colidx.shape[0])

    def copy(self) -> "HostBSR":
        return HostBSR(self.nbrows, self.nbcols, self.bs_r, self.bs_c, self.rowptr.copy(), self.colidx.copy(),
                       self.vals.copy())

    def to_scipy(self):
        import scipy.sparse as sp
        return sp.bsr_matrix((self.vals, self.colidx, self.rowptr),
                             shape=(self.nbrows * self.bs_r, self.nbcols * self.bs_c))

    def to_dense(self) -> np.ndarray:
        return np.asarray(self.to_scipy().todense())


# BASELINE.json configs: (dimension, elements per side, seed, modulus mode, number of levels)
CONFIGS = {
    0: dict(d=3, ne=8, seed=0, modulus_mode=0, nlevels=2, name="cfg0: 3D 8^3 Q1 hex elasticity, bs 3->6"),
    1: dict(d=2, ne=512, seed=1, modulus_mode=0, nlevels=2, name="cfg1: 2D 512^2 Q1 quad plane strain, bs 2->3"),
    2: dict(d=3, ne=64, seed=2, modulus_mode=0, nlevels=2, name="cfg2: 3D 64^3 Q1 hex elasticity, bs 3->6"),
    3: dict(d=3, ne=128, seed=3, modulus_mode=1, nlevels=2,
            name="cfg3: 3D 128^3 Q1 hex elasticity, lognormal E, bs 3->6"),
    4: dict(d=3, ne=96, seed=4, modulus_mode=0, nlevels=3, name="cfg4: 3D 96^3 Q1 hex elasticity, 3 levels"),
    # second workload: the same 65^3 node grid as config 2
    5: dict(d=3, ne=32, seed=5, modulus_mode=0, nlevels=2, order=2,
            name="cfg5: 3D 32^3 Q2 hex elasticity (65^3 nodes, ~185 nnz/row), bs 3->6, box aggregates"),
    6: dict(d=3, ne=64, seed=6, modulus_mode=0, nlevels=2, agg_mode=1,
            name="cfg6: 3D 64^3 Q1 hex elasticity, greedy (MIS-like) aggregates, bs 3->6"),
}

# random streams (reading R12)
PURPOSE_POWER, PURPOSE_FINE, PURPOSE_COARSE, PURPOSE_RHS, PURPOSE_MODULI, PURPOSE_RESCALE = 0, 1, 2, 3, 4, 5


def uniform(seed: int, purpose: int, n: int, a: float = -1.0, b: float = 1.0) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().egen_uniform(seed, purpose, n, a, b, out.ctypes.data)
    return out


def element_matrix(d: int, h: float, E: float = 1.0, nu: float = 0.3, order: int = 1) -> np.ndarray:
    nd = d * (order + 1) ** d
    out = np.empty((nd, nd), dtype=np.float64)
    if _load().egen_element_matrix2(d, order, h, E, nu, out.ctypes.data) != 0:
        raise ValueError("bad dimension or order")
    return out


class Generator:
    """One elasticity hierarchy under construction.  Arrays returned are views into generator-owned memory;
    keep the Generator alive while they are in use."""

    def __init__(self, d: int, ne: int, seed: int = 0, modulus_mode: int = 0, nu: float = 0.3,
                 dirichlet: bool = True, order: int = 1, agg_mode: int = 0):
        self._lib = _load()
        self.d, self.ne, self.seed, self.order, self.agg_mode = d, ne, seed, order, agg_mode
        self._h = self._lib.egen_create2(d, ne, nu, seed, modulus_mode, 1 if dirichlet else 0, order, agg_mode)
        if not self._h:
            raise ValueError("egen_create failed")

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.egen_destroy(self._h)
            self._h = None

    def _matrix(self, level: int, which: int) -> HostBSR:
        nbr, nbc, br, bc = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
        nnzb = C.c_int64()
        rp, ci, va = C.POINTER(C.c_int32)(), C.POINTER(C.c_int32)(), C.POINTER(C.c_double)()
        rc = self._lib.egen_matrix(self._h, level, which, nbr, nbc, br, bc, nnzb, rp, ci, va)
        if rc != 0:
            raise RuntimeError(f"matrix not available (level {level}, which {which})")
        n = nnzb.value
        rowptr = np.ctypeslib.as_array(rp, shape=(nbr.value + 1,))
        colidx = np.ctypeslib.as_array(ci, shape=(max(n, 1),))[:n]
        vals = np.ctypeslib.as_array(va, shape=(max(n, 1) * br.value * bc.value,))[:n * br.value * bc.value]
        return HostBSR(nbr.value, nbc.value, br.value, bc.value, rowptr, colidx,
                       vals.reshape(n, br.value, bc.value))

    def A(self, level: int = 0) -> HostBSR:
        return self._matrix(level, 0)

    def P(self, level: int = 0) -> HostBSR:
        return self._matrix(level, 1)

    def P_tent(self, level: int = 0) -> HostBSR:
        return self._matrix(level, 2)

    def build_prolongator(self, level: int = 0) -> None:
        if self._lib.egen_build_prolongator(self._h, level) != 0:
            raise RuntimeError(self._lib.egen_error(self._h).decode())

    def set_operator(self, level: int, A: HostBSR) -> None:
        rp = np.ascontiguousarray(A.rowptr, dtype=np.int32)
        ci = np.ascontiguousarray(A.colidx, dtype=np.int32)
        va = np.ascontiguousarray(A.vals, dtype=np.float64)
        rc = self._lib.egen_set_operator(self._h, level, A.nbrows, A.bs_r, A.nnzb, rp.ctypes.data, ci.ctypes.data,
                                         va.ctypes.data)
        if rc != 0:
            raise RuntimeError(f"egen_set_operator failed ({rc})")

    @property
    def nelements(self) -> int:
        return self.ne ** self.d

    def element_stream(self, e0: int = 0, e1: int | None = None, values: bool = True):
        """Blocked COO contribution stream of elements [e0, e1): (brow, bcol, blocks (n, d, d)),
        4^d contributions per element in element order; the clamped face is folded into the blocks (R4)."""
        e1 = self.nelements if e1 is None else e1
        n = (e1 - e0) * (self.order + 1) ** (2 * self.d)
        brow, bcol = np.empty(n, dtype=np.int32), np.empty(n, dtype=np.int32)
        vals = np.empty((n, self.d, self.d)) if values else None
        rc = self._lib.egen_element_stream(self._h, e0, e1, brow.ctypes.data, bcol.ctypes.data,
                                           vals.ctypes.data if values else None)
        if rc != 0:
            raise ValueError(f"egen_element_stream failed ({rc})")
        return brow, bcol, vals

    def element_data(self):
        """(per-element moduli or None, reference element matrix for E = 1): inputs of the device-side emission."""
        em, ke = C.POINTER(C.c_double)(), C.POINTER(C.c_double)()
        self._lib.egen_element_data(self._h, em, ke)
        nd = self.d * (self.order + 1) ** self.d
        K = np.ctypeslib.as_array(ke, shape=(nd, nd)).copy()
        E = np.ctypeslib.as_array(em, shape=(self.nelements,)).copy() if em else None
        return E, K

    def level_info(self, level: int) -> dict:
        nn, bs, nb = C.c_int32(), C.c_int32(), C.c_int32()
        nx = (C.c_int32 * 3)()
        lam, om = C.c_double(), C.c_double()
        if self._lib.egen_level_info(self._h, level, nn, bs, nb, nx, lam, om) != 0:
            raise IndexError(level)
        return dict(nnodes=nn.value, bs=bs.value, nb=nb.value, nx=tuple(nx), lam=lam.value, omega=om.value)

    def level_arrays(self, level: int) -> dict:
        info = self.level_info(level)
        co, rf, ag = C.POINTER(C.c_double)(), C.POINTER(C.c_double)(), C.POINTER(C.c_int32)()
        self._lib.egen_level_arrays(self._h, level, co, rf, ag)
        n, d, nb = info["nnodes"], self.d, info["nb"]
        out = dict(coords=np.ctypeslib.as_array(co, shape=(n, d)))
        out["rfac"] = np.ctypeslib.as_array(rf, shape=(n, nb, nb)) if rf else None
        out["agg"] = np.ctypeslib.as_array(ag, shape=(n,)) if ag else None
        return out


def make_generator(cfg: int, **over) -> Generator:
    c = dict(CONFIGS[cfg])
    c.update(over)
    return Generator(c["d"], c["ne"], c["seed"], c["modulus_mode"], dirichlet=c.get("dirichlet", True),
                     order=c.get("order", 1), agg_mode=c.get("agg_mode", 0))
