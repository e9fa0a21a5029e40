"""GPU parity tests: the CUDA path through the C ABI against the CPU oracle, element by element on the same seeded
inputs (readings R5, R14, R18).  Tolerances: structure bit-exact; values and SpMV outputs
1e-12 blockwise (north_star); residual history 1e-8 (R18)."""
import ctypes as C

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr
from tests.util import blockwise_rel_err, vec_blockwise_rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def bsr():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_24748_b200 import bsr as m
    m.lib()
    return m


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.cpu().numpy()


def abs_copy(M):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, np.abs(M.vals))


def check_spmv(bsr, M, seed, trans=False):
    """GPU y = M x (or M^T x) against the oracle, blockwise relative to max(|y|, 1e-3 |M||x|) (tests/util.py)."""
    n_in = M.nbrows * M.bs_r if trans else M.nbcols * M.bs_c
    x = pr.uniform(seed, pr.PURPOSE_FINE, n_in)
    G = bsr.Bsr.from_host(M)
    if trans:
        y = host(G.spmv_t(dev(x)))
        ref, mag, bs = orc.spmv_t(M, x), orc.spmv_t(abs_copy(M), np.abs(x)), M.bs_c
    else:
        y = host(G.spmv(dev(x)))
        ref, mag, bs = orc.spmv(M, x), orc.spmv(abs_copy(M), np.abs(x)), M.bs_r
    err = vec_blockwise_rel_err(y, ref, bs, mag)
    assert err < TOL, (M.bs_r, M.bs_c, trans, err)
    return G


def small_problems():
    g3 = pr.make_generator(0); g3.build_prolongator(0)            # 3x3, 3x6, 6x3, 6x6
    g2 = pr.Generator(2, 40, seed=1); g2.build_prolongator(0)     # 2x2, 2x3, 3x2, 3x3
    g3b = pr.Generator(3, 13, seed=5); g3b.build_prolongator(0)   # ragged: 14 nodes per side, merged last box
    return {"cfg0": g3, "quad40": g2, "hex13": g3b}


@pytest.fixture(scope="module")
def probs():
    return small_problems()


@pytest.mark.parametrize("name", ["cfg0", "quad40", "hex13"])
def test_spmv_family(bsr, probs, name):
    g = probs[name]
    A, P = g.A(0), g.P(0)
    check_spmv(bsr, A, g.seed)                 # y = A x     (3x3 / 2x2)
    check_spmv(bsr, P, g.seed)                 # y = P x_c   (3x6 / 2x3)
    check_spmv(bsr, P, g.seed, trans=True)     # y = P^T x   (6x3 / 3x2 on the cached transpose)
    R = orc.transpose(P)
    check_spmv(bsr, pr.HostBSR(R.nbrows, R.nbcols, R.bs_r, R.bs_c, R.rowptr, R.colidx, R.vals), g.seed)
    Ac = orc.ptap(A, P)                        # coarse operator: 6x6 / 3x3
    check_spmv(bsr, pr.HostBSR(Ac.nbrows, Ac.nbcols, Ac.bs_r, Ac.bs_c, Ac.rowptr, Ac.colidx, Ac.vals), g.seed)


def test_spmv_edge_structures(bsr):
    import torch
    rng = np.random.default_rng(3)
    for (br, bc) in [(2, 2), (2, 3), (3, 2), (3, 3), (3, 6), (6, 3), (6, 6)]:
        # empty rows, one-block rows, a 70-block row, odd nnzb; random columns
        lens = [0, 1, 0, 3, 70, 2, 0, 5, 1, 33, 0]
        nbcols = 90
        rowptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        cols = np.concatenate([np.sort(rng.choice(nbcols, n, replace=False)) for n in lens]).astype(np.int32)
        vals = rng.uniform(-1, 1, (cols.shape[0], br, bc))
        M = pr.HostBSR(len(lens), nbcols, br, bc, rowptr, cols, vals)
        assert M.nnzb % 2 == 1
        G = check_spmv(bsr, M, 9)
        check_spmv(bsr, M, 9, trans=True)
        # determinism: two runs give bit-identical outputs
        x = dev(pr.uniform(1, pr.PURPOSE_FINE, nbcols * bc))
        assert torch.equal(G.spmv(x), G.spmv(x))
    # empty matrix
    E = pr.HostBSR(0, 0, 3, 3, np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros((0, 3, 3)))
    G = bsr.Bsr.from_host(E)
    assert G.spmv(torch.empty(0, dtype=torch.float64, device="cuda")).numel() == 0


def test_spmv_flat_short_rows(bsr):
    """Short-row matrices of pair-able shapes take the flat value-stream kernel: many CTAs, empty rows, a ragged last
    CTA, rows of 1..8 blocks, and an all-empty matrix."""
    import torch
    rng = np.random.default_rng(11)
    for (br, bc) in [(3, 6), (2, 2), (6, 6)]:
        nbrows, nbcols = 1003, 400
        lens = rng.integers(0, 9, size=nbrows)
        lens[5:70] = 0                                           # a whole CTA's worth of empty rows
        if (br, bc) == (6, 6):
            lens = np.minimum(lens, 1)                           # keeps 6x6 in row mode (average below 2)
        rowptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        cols = np.concatenate([np.sort(rng.choice(nbcols, n, replace=False)) for n in lens] + [np.zeros(0, int)]).astype(np.int32)
        vals = rng.uniform(-1, 1, (cols.shape[0], br, bc))
        M = pr.HostBSR(nbrows, nbcols, br, bc, rowptr, cols, vals)
        G = check_spmv(bsr, M, 21)
        x = dev(pr.uniform(2, pr.PURPOSE_FINE, nbcols * bc))
        assert torch.equal(G.spmv(x), G.spmv(x))
    Z = pr.HostBSR(300, 10, 3, 6, np.zeros(301, np.int32), np.zeros(0, np.int32), np.zeros((0, 3, 6)))
    y = bsr.Bsr.from_host(Z).spmv(dev(np.ones(60)))
    assert float(y.abs().max()) == 0.0


def test_bsr_create_rejects_malformed(bsr):
    import torch
    ok = pr.HostBSR(2, 3, 3, 3, np.array([0, 2, 3], np.int32), np.array([0, 2, 1], np.int32), np.ones((3, 3, 3)))
    bsr.Bsr.from_host(ok)
    cases = {
        "unsorted": (np.array([0, 2, 3], np.int32), np.array([2, 0, 1], np.int32)),
        "duplicate": (np.array([0, 2, 3], np.int32), np.array([1, 1, 1], np.int32)),
        "range": (np.array([0, 2, 3], np.int32), np.array([0, 3, 1], np.int32)),
        "negative": (np.array([0, 2, 3], np.int32), np.array([-1, 2, 1], np.int32)),
        "monotone": (np.array([0, 3, 2], np.int32), np.array([0, 1, 2], np.int32)),
        "first": (np.array([1, 2, 3], np.int32), np.array([0, 1, 2], np.int32)),
        "last": (np.array([0, 2, 2], np.int32), np.array([0, 1, 2], np.int32)),
    }
    for name, (rp, ci) in cases.items():
        bad = pr.HostBSR(2, 3, 3, 3, rp, ci, np.ones((3, 3, 3)))
        with pytest.raises(bsr.BsrError) as e:
            bsr.Bsr.from_host(bad)
        assert e.value.code == 4, name
    with pytest.raises(bsr.BsrError) as e:
        bsr.Bsr(1, 1, 4, 4, torch.zeros(2, dtype=torch.int32, device="cuda"),
                torch.zeros(0, dtype=torch.int32, device="cuda"), torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert e.value.code == 3
    # misaligned vector pointer
    G = bsr.Bsr.from_host(ok)
    x = torch.zeros(10, dtype=torch.float64, device="cuda")[1:]
    with pytest.raises(bsr.BsrError) as e:
        G.spmv(x)
    assert e.value.code == 8


def ptap_check(bsr, A, P, Ac_ref=None):
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    plan = bsr.PtapPlan(GA, GP)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    assert np.array_equal(host(plan.rowptr_c), rc) and np.array_equal(host(plan.colidx_c), cc)   # bit exact
    vals = plan.numeric()
    rap_g, cap_g, ap_g = plan.ap_host()
    assert np.array_equal(rap_g, rap) and np.array_equal(cap_g, cap)
    if Ac_ref is None:
        Ac_ref = orc.ptap(A, P, structure=(rc, cc))
    mag = orc.ptap(abs_copy(A), abs_copy(P), structure=(rc, cc)).vals
    got = host(vals).reshape(-1, P.bs_c, P.bs_c)
    err = blockwise_rel_err(got, Ac_ref.vals, mag)
    assert err < TOL, err
    return GA, GP, plan, got, Ac_ref, mag


@pytest.mark.parametrize("name", ["cfg0", "quad40", "hex13"])
def test_ptap_structure_and_values(bsr, probs, name):
    g = probs[name]
    A, P = g.A(0), g.P(0)
    GA, GP, plan, got, ref, _ = ptap_check(bsr, A, P)
    # AP against the oracle's materialised AP (form 2)
    f2 = orc.PtapForm2(A, P)
    f2.run()
    f2m = orc.PtapForm2(abs_copy(A), abs_copy(P))
    f2m.run()
    _, _, ap = plan.ap_host()
    assert blockwise_rel_err(ap, f2.vals_ap, f2m.vals_ap) < TOL
    info = plan.info()
    assert info["nnzb_ap"] == f2.cap.shape[0]
    if name == "cfg0":
        assert (info["n_products_1"], info["n_products_2"]) == (50653, 15625)     # SURVEY.md master table


def test_ptap_recompute_reuse_and_state_gate(bsr, probs):
    """Config 2's protocol at config-0 size: ten recomputes over one plan, A rescaled per recompute (R13);
    closed form A_c^(k) = s_k A_c^(0) (pin I9); P-side cache rebuilt only when P's state moves;
    no allocation and no extra launches in the hot call."""
    import torch
    g = probs["cfg0"]
    A, P = g.A(0), g.P(0)
    GA, GP, plan, base, ref, mag = ptap_check(bsr, A, P)
    s = pr.uniform(2, pr.PURPOSE_RESCALE, 10, 0.5, 2.0)
    out = plan.new_values()
    assert plan.info()["n_r_value_builds"] == 1
    for sk in s:
        GA.set_values(A.vals * sk)
        l0, a0 = bsr.counters()
        plan.numeric(out)
        l1, a1 = bsr.counters()
        assert a1 == a0 and l1 - l0 == 2            # two kernels, no allocation, R not rebuilt
        got = host(out).reshape(base.shape)
        assert blockwise_rel_err(got, sk * ref.vals, sk * mag) < TOL       # oracle, closed form I9
        assert blockwise_rel_err(got, sk * base, sk * mag) < 1e-13         # and the GPU's own first result
    assert plan.info()["n_r_value_builds"] == 1
    # P changes: the gate opens exactly once
    GA.set_values(A.vals)
    GP.set_values(P.vals * 2.0)
    l0, _ = bsr.counters()
    plan.numeric(out)
    l1, _ = bsr.counters()
    assert l1 - l0 == 3 and plan.info()["n_r_value_builds"] == 2
    assert blockwise_rel_err(host(out).reshape(base.shape), 4.0 * base, 4.0 * mag) < 1e-14
    plan.numeric(out)
    assert plan.info()["n_r_value_builds"] == 2
    # determinism
    o2 = plan.numeric()
    assert torch.equal(out, o2)
    # a plan is bound to its matrices
    other = bsr.Bsr.from_host(A)
    with pytest.raises(bsr.BsrError) as e:
        bsr._check(bsr.lib().ptap_numeric(plan.h, other.h, GP.h, bsr._dev(out), 0))
    assert e.value.code == 7


def _random_bsr(rng, nbrows, nbcols, br, bc, row_len):
    lens = np.minimum(rng.integers(1, row_len + 1, size=nbrows), nbcols)
    rowptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    cols = np.concatenate([np.sort(rng.choice(nbcols, n, replace=False)) for n in lens]).astype(np.int32)
    return pr.HostBSR(nbrows, nbcols, br, bc, rowptr, cols, rng.uniform(-1, 1, (cols.shape[0], br, bc)))


def test_ptap_unstructured_falls_back_to_gather_kernels(bsr):
    """A product outside the staged format (AP / A_c rows with more than 32 blocks: random A and P) keeps the gather
    kernels; results must be the same definition."""
    rng = np.random.default_rng(5)
    A = _random_bsr(rng, 120, 120, 3, 3, 12)
    P = _random_bsr(rng, 120, 60, 3, 6, 9)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    assert np.diff(rap).max() > 32 or np.diff(rc).max() > 32
    ptap_check(bsr, A, P)


def test_ptap_gather_path_matches_staged_path(bsr, probs):
    """bsr_set_option("ptap_force_gather") keeps the one-thread-per-block gather kernels (the path a matrix outside
    the staged format takes) on a structured problem: same structure, values within rounding."""
    g = probs["hex13"]
    A, P = g.A(0), g.P(0)
    _, _, plan, staged, ref, mag = ptap_check(bsr, A, P)
    assert plan.schedule()[1]["staged"] == 1 and plan.schedule()[2]["staged"] == 1
    bsr.set_option("ptap_force_gather", 1)
    try:
        _, _, plan2, gathered, _, _ = ptap_check(bsr, A, P)
        assert plan2.schedule()[1]["staged"] == 0 and plan2.schedule()[2]["staged"] == 0
    finally:
        bsr.set_option("ptap_force_gather", 0)
    assert blockwise_rel_err(gathered, staged, mag) < 1e-13


def test_ptap_shape_errors(bsr, probs):
    g = probs["cfg0"]
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    with pytest.raises(bsr.BsrError) as e:
        bsr.PtapPlan(GP, GP)          # A not square
    assert e.value.code == 2
    g2 = probs["quad40"]
    with pytest.raises(bsr.BsrError) as e:
        bsr.PtapPlan(GA, bsr.Bsr.from_host(g2.P(0)))   # block sizes / sizes do not match
    assert e.value.code == 2


def test_spmv_host_end_to_end(bsr, probs):
    g = probs["cfg0"]
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    x = pr.uniform(0, pr.PURPOSE_FINE, A.nbrows * 3)
    y = np.empty(A.nbrows * 3)
    GA.spmv_host(x, y)
    assert vec_blockwise_rel_err(y, orc.spmv(A, x), 3, orc.spmv(abs_copy(A), np.abs(x))) < TOL
    yc = np.empty(P.nbcols * 6)
    GP.spmv_host(x, yc, trans=True)
    assert vec_blockwise_rel_err(yc, orc.spmv_t(P, x), 6, orc.spmv_t(abs_copy(P), np.abs(x))) < TOL
    # PtAP with host values in, host values out
    plan = bsr.PtapPlan(GA, GP)
    out = plan.new_values()
    h_out = np.empty(out.numel())
    plan.numeric_host(np.ascontiguousarray(A.vals * 1.5).reshape(-1), h_out, out)
    ref = orc.ptap(A, P)
    mag = orc.ptap(abs_copy(A), abs_copy(P)).vals
    assert blockwise_rel_err(h_out.reshape(ref.vals.shape), 1.5 * ref.vals, 1.5 * mag) < TOL


def test_workspace_comes_from_the_callers_allocator(bsr, probs):
    """Library workspace is obtained through bsr_set_allocator (torch's caching allocator in the harness), in cold
    calls only, and returned when the handles are destroyed; an allocator that fails surfaces as BSR_ERR_ALLOC."""
    import ctypes as C
    import torch
    g = probs["cfg0"]
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    w0 = bsr.workspace_bytes()
    plan = bsr.PtapPlan(GA, GP)
    w1 = bsr.workspace_bytes()
    assert w1 > w0 + plan.info()["nnzb_ap"] * 18 * 8            # at least AP's values live in torch memory now
    a0 = bsr.counters()[1]
    v = plan.numeric()
    assert bsr.counters()[1] == a0 and bsr.workspace_bytes() == w1   # hot call: no allocation
    plan.close(); GP.close()
    assert bsr.workspace_bytes() <= w0
    # a failing allocator: the cold call reports BSR_ERR_ALLOC and nothing leaks
    fail_alloc = bsr._ALLOC_FN(lambda n, ctx: None)
    noop_free = bsr._FREE_FN(lambda p, ctx: None)
    bsr._check(bsr.lib().bsr_set_allocator(C.cast(fail_alloc, C.c_void_p), C.cast(noop_free, C.c_void_p), None))
    try:
        GP2 = bsr.Bsr.from_host(P)
        with pytest.raises(bsr.BsrError) as e:
            bsr.PtapPlan(GA, GP2)
        assert e.value.code == 5
    finally:
        bsr.use_torch_allocator(True)
    plan2 = bsr.PtapPlan(GA, GP2)                               # and the library works again afterwards
    assert torch.equal(plan2.numeric(), v)


def test_ptap_host_buffer_path_is_chunked_and_exact(bsr, probs):
    """ptap_numeric_host: A's values arrive from a HOST buffer in row chunks on a copy stream, stage 1 runs behind the
    chunks, A_c leaves in pieces behind stage 2 -- the result must be bit-identical to ptap_numeric on device values,
    call after call with changing values."""
    import torch
    for name in ("hex13", "quad40", "cfg0"):
        g = probs[name]
        A, P = g.A(0), g.P(0)
        GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
        plan = bsr.PtapPlan(GA, GP)
        vals_c = plan.new_values()
        hc = torch.empty(vals_c.numel(), dtype=torch.float64).pin_memory()
        for k, scale in enumerate((1.0, 0.37, 2.5)):
            ha = torch.from_numpy(np.ascontiguousarray(A.vals.reshape(-1) * scale)).pin_memory()
            plan.numeric_host(ha.numpy(), hc.numpy(), vals_c)
            GA2 = bsr.Bsr.from_host(pr.HostBSR(A.nbrows, A.nbcols, A.bs_r, A.bs_c, A.rowptr, A.colidx, A.vals * scale))
            ref = bsr.PtapPlan(GA2, GP).numeric()
            assert torch.equal(vals_c, ref), (name, k)
            assert np.array_equal(hc.numpy(), ref.cpu().numpy()), (name, k)
            assert np.array_equal(GA.vals.cpu().numpy(), ha.numpy())        # the device copy of A holds the new values


def test_fp64_peak_probes(bsr):
    """The two ALU roofs bench.py reports: FMA chains and mma.sync m8n8k4 chains.  On B200 both land near 37 TFLOP/s;
    the test only pins that they are positive, of the same order, and below what 148 SMs x 128 FMA/clk x 2.5 GHz allow."""
    fma = bsr.fp64_peak_tflops()
    mma = bsr.fp64_peak_tflops(mma=True)
    assert 1.0 < fma < 100.0 and 1.0 < mma < 100.0
    assert 0.5 < mma / fma < 2.0
