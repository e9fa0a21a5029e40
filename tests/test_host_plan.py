"""CPU tests of the library's host logic (no GPU): symbol table, error paths that need no device, and the
symbolic plan of ptap_symbolic checked against the oracle (structure bit-exact; the plan's product lists evaluated
in numpy reproduce the oracle's AP and A_c)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import bsr
from paper_2606_24748_b200 import problems as pr
from tests.util import blockwise_rel_err

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "bsr_amg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b((?:bsr|ptap|vcycle|pcg|prolongator_smooth|bcoo|fem_q1)_[a-z_0-9]+)\s*\(", hdr))
    assert {"bsr_create", "bsr_spmv", "bsr_spmv_t", "ptap_symbolic", "ptap_numeric", "vcycle_apply"} <= declared
    L = bsr.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(bsr.SYMBOLS), declared ^ set(bsr.SYMBOLS)


def test_null_and_shape_errors_without_device():
    L = bsr.lib()
    h = C.c_void_p()
    assert L.bsr_create(None, 1, 1, 3, 3, 0, None, None, None, None) == 1
    assert L.bsr_create(C.byref(h), 1, 1, 3, 3, 0, None, None, None, None) == 1  # null rowptr
    dummy = (C.c_int32 * 4)()
    dvals = (C.c_double * 64)()
    assert L.bsr_create(C.byref(h), 1, 1, 4, 4, 1, dummy, dummy, dvals, None) == 3  # 4x4 unsupported
    assert b"4x4" in L.bsr_last_error()
    assert L.bsr_create(C.byref(h), -1, 1, 3, 3, 0, dummy, dummy, dvals, None) == 2
    assert L.bsr_spmv(None, None, None, None) == 1
    assert L.bsr_spmv_t(None, None, None, None) == 1
    assert L.ptap_numeric(None, None, None, None, None) == 1
    assert L.vcycle_apply(None, None, None, None) == 1
    assert L.pcg_solve(None, None, None, 1, None, None) == 1
    assert L.bsr_destroy(None) == 0 and L.ptap_destroy(None) == 0 and L.vcycle_destroy(None) == 0
    assert L.ptap_host_plan_build(1, None, None, 1, None, None) is None


def _eval_stage(pairptr, ox, oy, rowidx, rowptr_x, ystart, X, Y):
    """Evaluate the gather plan in numpy: out[u] = sum_p X[x0 + ox[p]] @ Y[ystart[x0 + ox[p]] + oy[p]]."""
    n = pairptr.shape[0] - 1
    out = np.zeros((n, X.shape[1], Y.shape[2]))
    seg = np.repeat(np.arange(n), np.diff(pairptr))
    xs = rowptr_x[rowidx[seg]] + ox.astype(np.int64)
    ys = ystart[xs] + oy.astype(np.int64)
    prod = np.einsum("prk,pkc->prc", X[xs], Y[ys])
    np.add.at(out, seg, prod)
    return out, xs


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_host_plan_matches_oracle(fix, request):
    g = request.getfixturevalue(fix)
    A, P = g.A(0), g.P(0)
    hp = bsr.HostPlan(A, P)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    R = orc.transpose(P)
    # structures: bit exact
    assert np.array_equal(hp.rowptr_ap, rap) and np.array_equal(hp.colidx_ap, cap)
    assert np.array_equal(hp.rowptr_c, rc) and np.array_equal(hp.colidx_c, cc)
    assert np.array_equal(hp.rowptr_r, R.rowptr) and np.array_equal(hp.colidx_r, R.colidx)
    assert np.array_equal(P.vals[hp.perm_r].transpose(0, 2, 1), R.vals)
    assert np.array_equal(hp.rowidx_ap, np.repeat(np.arange(A.nbrows), np.diff(rap)))
    assert np.array_equal(hp.rowidx_c, np.repeat(np.arange(P.nbcols), np.diff(rc)))
    # product lists: ascending inner index inside each output block, and they reproduce the oracle's values
    ap, xs1 = _eval_stage(hp.pairptr1, hp.k1, hp.q1, hp.rowidx_ap, A.rowptr, hp.pstart, A.vals, P.vals)
    for s in range(0, hp.pairptr1.shape[0] - 1, 7):
        seg = xs1[hp.pairptr1[s]:hp.pairptr1[s + 1]]
        assert (np.diff(seg) > 0).all()
    f2 = orc.PtapForm2(A, P)
    Ac_o = f2.run()
    # blocks that cancel to rounding level are measured against their magnitude sum |A||P| (tests/util.py)
    s_ap, _ = _eval_stage(hp.pairptr1, hp.k1, hp.q1, hp.rowidx_ap, A.rowptr, hp.pstart, np.abs(A.vals), np.abs(P.vals))
    assert blockwise_rel_err(ap, f2.vals_ap, s_ap) < 1e-13
    ac, _ = _eval_stage(hp.pairptr2, hp.t2, hp.s2, hp.rowidx_c, hp.rowptr_r, hp.apstart, R.vals, ap)
    s_ac, _ = _eval_stage(hp.pairptr2, hp.t2, hp.s2, hp.rowidx_c, hp.rowptr_r, hp.apstart, np.abs(R.vals), s_ap)
    assert blockwise_rel_err(ac, orc.ptap(A, P).vals, s_ac) < 1e-12
    assert blockwise_rel_err(ac, Ac_o.vals, s_ac) < 1e-12
    # counts of SURVEY.md's master table at config 0
    if fix == "cfg0":
        assert hp.colidx_ap.shape[0] == 4913 and hp.colidx_c.shape[0] == 343
        assert hp.k1.shape[0] == 50653 and hp.t2.shape[0] == 15625


def test_host_plan_rejects_nothing_silently_on_empty_rows():
    # a matrix with empty rows and an empty P column: structures stay consistent
    A = pr.HostBSR(3, 3, 3, 3, np.array([0, 1, 1, 2], np.int32), np.array([0, 2], np.int32), np.ones((2, 3, 3)))
    P = pr.HostBSR(3, 2, 3, 6, np.array([0, 1, 1, 2], np.int32), np.array([0, 0], np.int32), np.ones((2, 3, 6)))
    hp = bsr.HostPlan(A, P)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    assert np.array_equal(hp.rowptr_ap, rap) and np.array_equal(hp.colidx_ap, cap)
    assert np.array_equal(hp.rowptr_c, rc) and np.array_equal(hp.colidx_c, cc)
    assert hp.rowptr_c.tolist() == [0, 1, 1]


def test_staged_schedule_covers_every_product_once():
    """Host logic of the staged numeric PtAP (ptap_stream.cpp): the per-block masks of both stages must hold exactly
    one bit per block product of the gather plan, every brick must fit its shared-memory budget, and stage 2 has one
    brick per coarse row."""
    from paper_2606_24748_b200 import bsr, problems as pr
    for g in (pr.make_generator(0), pr.Generator(2, 24, seed=3), pr.Generator(3, 13, seed=5)):
        g.build_prolongator(0)
        A, P = g.A(0), g.P(0)
        hp = bsr.HostPlan(A, P)
        s1, s2 = hp.stream_stats[1], hp.stream_stats[2]
        assert s1["ok"] == 1 and s2["ok"] == 1
        assert s1["mask_bits"] == hp.k1.shape[0]          # stage 1: every A(i,j)*P(j,J) product once
        assert s2["mask_bits"] == hp.t2.shape[0]          # stage 2: every R(I,i)*AP(i,K) product once
        assert s1["max_smem"] <= 112 * 1024 and s2["max_smem"] <= 75000
        assert s2["bricks"] == P.nbcols and s2["chunks"] >= s2["bricks"]
        assert s1["lanes"] == hp.colidx_ap.shape[0]       # one lane per AP block
        assert s1["passes"] * 32 >= s1["lanes"] and s1["steps"] > 0


def test_limit_errors_without_device():
    """BSR_ERR_LIMIT: 32-bit counts that would overflow are refused before any device work."""
    L = bsr.lib()
    h = C.c_void_p()
    fake = C.c_void_p(256)                                   # never dereferenced: the size check comes first
    nnzb = (1 << 31) // 9 + 1
    rc = L.bsr_create(C.byref(h), 10, 10, 3, 3, nnzb, fake, fake, fake, None)
    assert rc == 10 and b"2^31" in L.bsr_last_error() and not h.value
    nn = C.c_int64()
    rc = L.bcoo_plan_create(C.byref(h), 1 << 31, fake, fake, 10, 10, 3, 3, C.byref(nn), None)
    assert rc == 10 and not h.value
    rc = L.bsr_gather_blocks(1 << 40, fake, 9, fake, fake, None)
    assert rc == 10
    # the allocator registration wants both callbacks or neither
    assert L.bsr_set_allocator(fake, None, None) == 1
    assert L.bsr_set_allocator(None, None, None) == 0
