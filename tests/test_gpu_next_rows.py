"""GPU parity of SURVEY.md 8(f) rows f1 (device prolongator smoothing) and f2 (blocked COO assembly, driven by Q1
finite-element contributions) against the oracle (oracle/oracle.cpp: orc_prolongator_smooth, orc_bcoo_*), element by
element: structure arrays with ==, values blockwise at 1e-12 (north_star), at small sizes that span several bricks and
ragged tails, and at BASELINE.json's full sizes (every block at configs 1-4 for f1; config 2 complete and a seeded
element slab at config 3 for f2, where the oracle's long-double accumulators for the whole grid would need tens of GB).
All calls go through the C ABI (paper_2606_24748_b200/bsr.py marshals only)."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr
from tests.util import blockwise_rel_err

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


def as_host(M, vals=None):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, M.vals if vals is None else vals)


# ------------------------------------------------------------------ f1: prolongator smoothing
def smooth_check(bsr, A, Pt, omega, expect_staged=None):
    GA, GT = bsr.Bsr.from_host(A), bsr.Bsr.from_host(Pt)
    sm = bsr.ProlongatorSmoother(GA, GT)
    ref = orc.prolongator_smooth(A, Pt, omega)
    assert np.array_equal(sm.rowptr_p.cpu().numpy(), ref.rowptr) and np.array_equal(sm.colidx_p.cpu().numpy(), ref.colidx)
    if expect_staged is not None:
        assert sm.info()["staged"] == expect_staged
    a0 = bsr.counters()[1]
    vals = sm.numeric(omega, check=True)
    assert bsr.counters()[1] == a0                                     # hot: no allocation
    got = vals.cpu().numpy().reshape(ref.vals.shape)
    err = blockwise_rel_err(got, ref.vals)
    assert err < TOL, err
    import torch
    assert torch.equal(vals, sm.numeric(omega))                         # bit-reproducible
    return sm, GA, GT, vals, ref


def level2_problem(d, ne, seed):
    g = pr.Generator(d, ne, seed=seed)
    g.build_prolongator(0)
    Ac = orc.ptap(g.A(0), g.P(0))
    A1 = as_host(Ac)
    g.set_operator(1, A1)
    g.build_prolongator(1)
    return g, A1


@pytest.mark.parametrize("name", ["cfg0", "quad40", "hex13", "level2_6x6", "level2_3x3"])
def test_prolongator_smooth_small(bsr, name):
    if name == "cfg0":
        g = pr.make_generator(0); g.build_prolongator(0); A, Pt, om = g.A(0), g.P_tent(0), g.level_info(0)["omega"]
    elif name == "quad40":
        g = pr.Generator(2, 40, seed=1); g.build_prolongator(0); A, Pt, om = g.A(0), g.P_tent(0), g.level_info(0)["omega"]
    elif name == "hex13":
        g = pr.Generator(3, 13, seed=2, modulus_mode=1); g.build_prolongator(0)
        A, Pt, om = g.A(0), g.P_tent(0), g.level_info(0)["omega"]
    elif name == "level2_6x6":
        g, A = level2_problem(3, 11, 4); Pt, om = g.P_tent(1), g.level_info(1)["omega"]
    else:
        g, A = level2_problem(2, 33, 5); Pt, om = g.P_tent(1), g.level_info(1)["omega"]
    sm, GA, GT, vals, ref = smooth_check(bsr, A, Pt, om, expect_staged=True)
    # the generator's host loop gives the same P: the device-built prolongator can replace it
    lvl = 1 if name.startswith("level2") else 0
    assert np.abs(vals.cpu().numpy().reshape(ref.vals.shape) - g.P(lvl).vals).max() < 1e-13
    # omega = 0 returns P~ on the wider pattern exactly
    v0 = sm.numeric(0.0).cpu().numpy().reshape(ref.vals.shape)
    own = orc.prolongator_smooth(A, Pt, 0.0).vals
    assert np.array_equal(v0, own)
    # the gather fallback computes the same values
    bsr.set_option("ptap_force_gather", 1)
    try:
        smooth_check(bsr, A, Pt, om, expect_staged=False)
    finally:
        bsr.set_option("ptap_force_gather", 0)


@pytest.mark.parametrize("name", ["cfg0", "quad40", "level2_6x6", "cfg2"])
def test_power_iteration_lambda_on_device(bsr, name):
    """The eigenvalue estimate behind omega (reading R10) on the device against the oracle's power iteration; with it
    new A -> omega -> new P needs no host arithmetic."""
    if name == "cfg0":
        g = pr.make_generator(0); g.build_prolongator(0); A, Pt, lvl = g.A(0), g.P_tent(0), 0
    elif name == "quad40":
        g = pr.Generator(2, 40, seed=1); g.build_prolongator(0); A, Pt, lvl = g.A(0), g.P_tent(0), 0
    elif name == "level2_6x6":
        g, A = level2_problem(3, 11, 4); Pt, lvl = g.P_tent(1), 1
    else:
        g = pr.make_generator(2); g.build_prolongator(0); A, Pt, lvl = g.A(0), g.P_tent(0), 0
    v0 = pr.uniform(g.seed, pr.PURPOSE_POWER + 16 * lvl, A.nbrows * A.bs_r)
    GA, GT = bsr.Bsr.from_host(A), bsr.Bsr.from_host(Pt)
    sm = bsr.ProlongatorSmoother(GA, GT)
    lam = sm.lambda_estimate(dev(v0), 20)
    ref = orc.power_lambda(A, v0, 20)
    assert abs(lam / ref - 1) < 1e-11, (lam, ref)
    assert abs(lam / g.level_info(lvl)["lam"] - 1) < 1e-11           # = the generator's estimate
    assert lam == sm.lambda_estimate(dev(v0), 20)                    # fixed summation order: bit-reproducible
    # omega from the device estimate gives the oracle's P
    om = 4.0 / (3.0 * lam)
    got = sm.numeric(om, check=True).cpu().numpy()
    refP = orc.prolongator_smooth(A, Pt, 4.0 / (3.0 * ref))
    assert blockwise_rel_err(got.reshape(refP.vals.shape), refP.vals) < 1e-11


def test_ptap_on_device_built_prolongator(bsr):
    """New A -> new P -> new A_c without the host: smooth on the device, then ptap_numeric on that P."""
    g = pr.Generator(3, 12, seed=6, modulus_mode=1)
    g.build_prolongator(0)
    A, Pt, om = g.A(0), g.P_tent(0), g.level_info(0)["omega"]
    sm, GA, GT, vals, ref = smooth_check(bsr, A, Pt, om)
    GP = sm.matrix(vals)
    plan = bsr.PtapPlan(GA, GP)
    vc = plan.numeric()
    Pd = as_host(ref, vals.cpu().numpy().reshape(ref.vals.shape))       # the oracle multiplies the GPU's own P
    Ac = orc.ptap(A, Pd)
    mag = orc.ptap(as_host(A, np.abs(A.vals)), as_host(Pd, np.abs(Pd.vals)), structure=(Ac.rowptr, Ac.colidx)).vals
    assert np.array_equal(plan.rowptr_c.cpu().numpy(), Ac.rowptr) and np.array_equal(plan.colidx_c.cpu().numpy(), Ac.colidx)
    assert blockwise_rel_err(vc.cpu().numpy().reshape(Ac.vals.shape), Ac.vals, mag) < TOL
    # A changes, P~ does not: re-smooth in place and recompute (the state gate sees the new P)
    GA.vals.mul_(1.7); GA.values_changed()
    sm.numeric(om, vals); GP.values_changed()
    got = vals.cpu().numpy().reshape(ref.vals.shape)
    assert blockwise_rel_err(got, orc.prolongator_smooth(as_host(A, 1.7 * A.vals), Pt, om).vals) < TOL
    plan.numeric(vc)
    Pd2 = as_host(ref, got)
    Ac2 = orc.ptap(as_host(A, 1.7 * A.vals), Pd2)
    mag2 = orc.ptap(as_host(A, np.abs(1.7 * A.vals)), as_host(Pd2, np.abs(got)), structure=(Ac.rowptr, Ac.colidx)).vals
    assert blockwise_rel_err(vc.cpu().numpy().reshape(Ac.vals.shape), Ac2.vals, mag2) < TOL


def test_prolongator_smooth_errors(bsr):
    g = pr.make_generator(0); g.build_prolongator(0)
    A, Pt, P = g.A(0), g.P_tent(0), g.P(0)
    GA, GT, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(Pt), bsr.Bsr.from_host(P)
    with pytest.raises(bsr.BsrError) as e:
        bsr.ProlongatorSmoother(GT, GT)                                  # A not square
    assert e.value.code == 2
    sm = bsr.ProlongatorSmoother(GA, GT)
    sm2 = bsr.ProlongatorSmoother(GA, GP)
    out = sm.new_values()
    with pytest.raises(bsr.BsrError) as e:                               # plan used with another P~
        bsr._check(bsr.lib().prolongator_smooth_numeric(sm.h, GA.h, GP.h, 0.5, bsr._dev(out), 0))
    assert e.value.code == 7
    with pytest.raises(bsr.BsrError) as e:                               # misaligned output
        bsr._check(bsr.lib().prolongator_smooth_numeric(sm.h, GA.h, GT.h, 0.5, out.data_ptr() + 8, 0))
    assert e.value.code == 8
    # a row without its diagonal block whose own aggregate is still reached through a neighbour: numeric error
    keep = np.ones(A.nnzb, bool)
    keep[np.searchsorted(A.colidx[A.rowptr[5]:A.rowptr[6]], 5) + A.rowptr[5]] = False
    rp = A.rowptr.copy(); rp[6:] -= 1
    Abad = pr.HostBSR(A.nbrows, A.nbcols, 3, 3, rp, A.colidx[keep], A.vals[keep])
    smb = bsr.ProlongatorSmoother(bsr.Bsr.from_host(Abad), GT)
    with pytest.raises(bsr.BsrError) as e:
        smb.numeric(0.5, check=True)
    assert e.value.code == 9
    # no diagonal blocks at all: a P~ block falls outside the pattern of A*P~
    A2 = pr.HostBSR(2, 2, 2, 2, np.array([0, 1, 2], np.int32), np.array([1, 0], np.int32), np.ones((2, 2, 2)))
    T2 = pr.HostBSR(2, 2, 2, 3, np.array([0, 1, 2], np.int32), np.array([0, 1], np.int32), np.ones((2, 2, 3)))
    with pytest.raises(bsr.BsrError) as e:
        bsr.ProlongatorSmoother(bsr.Bsr.from_host(A2), bsr.Bsr.from_host(T2))
    assert e.value.code == 4
    # a singular diagonal block is reported by the status call
    GA.vals.zero_(); GA.values_changed()
    with pytest.raises(bsr.BsrError) as e:
        sm.numeric(0.5, check=True)
    assert e.value.code == 9
    del sm2


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_prolongator_smooth_full_size(bsr, cfg):
    """Every block of P at the BASELINE.json sizes (config 4: both levels)."""
    g = pr.make_generator(cfg)
    g.build_prolongator(0)
    A, Pt, om = g.A(0), g.P_tent(0), g.level_info(0)["omega"]
    sm, GA, GT, vals, ref = smooth_check(bsr, A, Pt, om, expect_staged=True)
    assert sm.nnzb_p == g.P(0).nnzb
    if cfg == 4:
        GP = sm.matrix(vals)
        plan = bsr.PtapPlan(GA, GP)
        v1 = plan.numeric()
        A1 = pr.HostBSR(plan.nbrows_c, plan.nbrows_c, 6, 6, plan.rowptr_c.cpu().numpy(), plan.colidx_c.cpu().numpy(),
                        v1.cpu().numpy().reshape(-1, 6, 6))
        g.set_operator(1, A1)
        g.build_prolongator(1)
        smooth_check(bsr, A1, g.P_tent(1), g.level_info(1)["omega"], expect_staged=True)


# ------------------------------------------------------------------ f2: blocked COO assembly
@pytest.mark.parametrize("br,bc", [(2, 2), (2, 3), (3, 2), (3, 3), (3, 6), (6, 3), (6, 6)])
def test_bcoo_random_coordinates(bsr, br, bc):
    import torch
    rng = np.random.default_rng(100 * br + bc)
    nbrows, nbcols, n = 301, 257, 20011
    brow = rng.integers(0, nbrows, n).astype(np.int32)
    bcol = rng.integers(0, nbcols, n).astype(np.int32)
    brow[:500] = 17; bcol[:500] = rng.integers(0, 5, 500)               # a long duplicate segment
    keep = brow != 100                                                  # an empty row
    brow, bcol = brow[keep], bcol[keep]
    stream = rng.uniform(-1, 1, (brow.shape[0], br, bc))
    ref = orc.bcoo_assemble(brow, bcol, stream, nbrows, nbcols)
    plan = bsr.BcooPlan(dev(brow), dev(bcol), nbrows, nbcols, br, bc)
    assert np.array_equal(plan.rowptr.cpu().numpy(), ref.rowptr) and np.array_equal(plan.colidx.cpu().numpy(), ref.colidx)
    a0 = bsr.counters()[1]
    vals = plan.set_values(dev(stream.reshape(-1)))
    assert bsr.counters()[1] == a0
    mag = orc.bcoo_assemble(brow, bcol, np.abs(stream), nbrows, nbcols, structure=(ref.rowptr, ref.colidx)).vals
    assert blockwise_rel_err(vals.cpu().numpy().reshape(ref.vals.shape), ref.vals, mag) < TOL
    assert torch.equal(vals, plan.set_values(dev(stream.reshape(-1))))   # bit-reproducible
    # a second stream through the same plan (the plan is reused; values only change)
    s2 = rng.uniform(-1, 1, stream.shape)
    ref2 = orc.bcoo_assemble(brow, bcol, s2, nbrows, nbcols, structure=(ref.rowptr, ref.colidx))
    mag2 = orc.bcoo_assemble(brow, bcol, np.abs(s2), nbrows, nbcols, structure=(ref.rowptr, ref.colidx)).vals
    assert blockwise_rel_err(plan.set_values(dev(s2.reshape(-1)), vals).cpu().numpy().reshape(ref.vals.shape),
                             ref2.vals, mag2) < TOL
    # the assembled matrix is a valid library matrix (bsr_create's validation accepts the structure)
    M = plan.matrix(vals)
    x = rng.uniform(-1, 1, nbcols * bc)
    y = M.spmv(dev(x)).cpu().numpy()
    assert np.abs(y - orc.spmv(as_host(ref2, vals.cpu().numpy().reshape(ref.vals.shape)), x)).max() < 1e-11


def test_bcoo_edge_cases(bsr):
    import torch
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    plan = bsr.BcooPlan(e, e, 5, 5, 3, 3)                                # no contribution at all
    assert plan.nnzb == 0 and plan.rowptr.cpu().tolist() == [0] * 6
    plan.set_values(torch.empty(0, dtype=torch.float64, device="cuda"))
    with pytest.raises(bsr.BsrError) as ex:                              # coordinate out of range
        bsr.BcooPlan(dev(np.array([0, 5], np.int32)), dev(np.array([0, 0], np.int32)), 5, 5, 3, 3)
    assert ex.value.code == 4
    with pytest.raises(bsr.BsrError) as ex:                              # unsupported block shape
        bsr.BcooPlan(dev(np.array([0], np.int32)), dev(np.array([0], np.int32)), 5, 5, 4, 4)
    assert ex.value.code == 3
    one = bsr.BcooPlan(dev(np.array([2] * 7, np.int32)), dev(np.array([3] * 7, np.int32)), 5, 5, 2, 3)
    s = np.arange(42, dtype=np.float64).reshape(7, 2, 3)
    assert np.array_equal(one.set_values(dev(s.reshape(-1))).cpu().numpy().reshape(2, 3), s.sum(axis=0))


def test_bcoo_block_larger_than_a_cta(bsr):
    """One destination block with more contributions than a CTA of the staged kernel parks (8192 doubles): the plan falls
    back to the per-value kernel for the whole matrix; same sums in the same order."""
    rng = np.random.default_rng(5)
    n_big = 3000
    brow = np.concatenate([np.full(n_big, 4), rng.integers(0, 9, 400)]).astype(np.int32)
    bcol = np.concatenate([np.full(n_big, 2), rng.integers(0, 9, 400)]).astype(np.int32)
    order = rng.permutation(brow.shape[0])
    brow, bcol = brow[order], bcol[order]
    stream = rng.uniform(-1, 1, (brow.shape[0], 3, 3))
    ref = orc.bcoo_assemble(brow, bcol, stream, 9, 9)
    plan = bsr.BcooPlan(dev(brow), dev(bcol), 9, 9, 3, 3)
    assert np.array_equal(plan.rowptr.cpu().numpy(), ref.rowptr) and np.array_equal(plan.colidx.cpu().numpy(), ref.colidx)
    vals = plan.set_values(dev(stream.reshape(-1))).cpu().numpy().reshape(ref.vals.shape)
    mag = orc.bcoo_assemble(brow, bcol, np.abs(stream), 9, 9, structure=(ref.rowptr, ref.colidx)).vals
    assert blockwise_rel_err(vals, ref.vals, mag) < TOL


def fem_device_assembly(bsr, g, chunk=None):
    """Config's operator assembled on the device: coordinates and E_e * Ke blocks emitted by the library's Q1 driver,
    summed through the blocked COO plan."""
    d, ne = g.d, g.ne
    E, Ke = g.element_data()
    dKe, dE = dev(Ke.reshape(-1)), (dev(E) if E is not None else None)
    nel = g.nelements
    brow, bcol = bsr.fem_q1_coords(d, ne, 0, nel)
    n = (ne + 1) ** d
    plan = bsr.BcooPlan(brow, bcol, n, n, d, d)
    stream = bsr.fem_q1_blocks(d, ne, 0, nel, dKe, dE, True)
    vals = plan.set_values(stream)
    return plan, vals, brow, bcol, stream


@pytest.mark.parametrize("d,ne,mode", [(3, 8, 0), (2, 40, 1), (3, 13, 1)])
def test_fem_assembly_small(bsr, d, ne, mode):
    g = pr.Generator(d, ne, seed=3, modulus_mode=mode)
    A = g.A(0)
    plan, vals, brow, bcol, stream = fem_device_assembly(bsr, g)
    hb, hc, hv = g.element_stream()
    assert np.array_equal(brow.cpu().numpy(), hb) and np.array_equal(bcol.cpu().numpy(), hc)
    assert np.array_equal(stream.cpu().numpy().reshape(hv.shape), hv)        # one multiplication per value: bit-equal
    ref = orc.bcoo_assemble(hb, hc, hv, A.nbrows, A.nbcols)
    assert np.array_equal(plan.rowptr.cpu().numpy(), ref.rowptr) and np.array_equal(plan.colidx.cpu().numpy(), ref.colidx)
    assert np.array_equal(ref.rowptr, A.rowptr) and np.array_equal(ref.colidx, A.colidx)
    mag = orc.bcoo_assemble(hb, hc, np.abs(hv), A.nbrows, A.nbcols, structure=(ref.rowptr, ref.colidx)).vals
    got = vals.cpu().numpy().reshape(ref.vals.shape)
    assert blockwise_rel_err(got, ref.vals, mag) < TOL
    assert blockwise_rel_err(got, A.vals, mag) < TOL                         # = the generator's gather-form assembly


def test_fem_assembly_config2_complete(bsr):
    g = pr.make_generator(2)
    A = g.A(0)
    plan, vals, brow, bcol, stream = fem_device_assembly(bsr, g)
    assert plan.n == 64 ** 3 * 64 and plan.nnzb == A.nnzb == 7189057
    hb, hc, hv = g.element_stream()
    ref = orc.bcoo_assemble(hb, hc, hv, A.nbrows, A.nbcols)
    assert np.array_equal(plan.rowptr.cpu().numpy(), ref.rowptr) and np.array_equal(plan.colidx.cpu().numpy(), ref.colidx)
    mag = orc.bcoo_assemble(hb, hc, np.abs(hv), A.nbrows, A.nbcols, structure=(ref.rowptr, ref.colidx)).vals
    got = vals.cpu().numpy().reshape(ref.vals.shape)
    assert blockwise_rel_err(got, ref.vals, mag) < TOL
    assert np.array_equal(ref.rowptr, A.rowptr) and blockwise_rel_err(got, A.vals, mag) < TOL


def test_fem_assembly_config3_headline_grid(bsr):
    """128^3, lognormal modulus: the whole operator is assembled on the device (134 M block contributions); structure
    and values are compared with the generator's operator over the whole matrix, and with the oracle on a seeded
    slab of element planes (rows of the nodes strictly inside the slab receive all their contributions from it)."""
    import torch
    g = pr.make_generator(3)
    A = g.A(0)
    plan, vals, brow, bcol, stream = fem_device_assembly(bsr, g)
    assert plan.n == 128 ** 3 * 64 and plan.nnzb == A.nnzb == 57066625
    assert np.array_equal(plan.rowptr.cpu().numpy(), A.rowptr) and np.array_equal(plan.colidx.cpu().numpy(), A.colidx)
    got = vals.cpu().numpy().reshape(A.vals.shape)
    del stream
    # whole matrix against the generator (gather-form host assembly, same addition order)
    scale = np.abs(A.vals).reshape(A.nnzb, -1).max(axis=1)
    dn = np.abs(got - A.vals).reshape(A.nnzb, -1).max(axis=1)
    assert (dn <= 1e-13 * np.maximum(scale, scale.max() * 1e-6)).all()
    print(f"[parity] cfg3 assembled A: {int((got == A.vals).all(axis=(1, 2)).sum())} of {A.nnzb} blocks bit-equal "
          f"to the host assembly")
    # oracle on element planes ez in [z0, z1): node planes z0+1 .. z1-1 are complete
    ne, n = 128, 129
    z0, z1 = 61, 65
    e0, e1 = z0 * ne * ne, z1 * ne * ne
    hb, hc, hv = g.element_stream(e0, e1)
    ref = orc.bcoo_assemble(hb, hc, hv, A.nbrows, A.nbcols)
    mag = orc.bcoo_assemble(hb, hc, np.abs(hv), A.nbrows, A.nbcols, structure=(ref.rowptr, ref.colidx)).vals
    rows = np.arange((z0 + 1) * n * n, z1 * n * n)
    for r0 in (rows[0], rows[-1]):
        assert ref.rowptr[r0 + 1] - ref.rowptr[r0] == A.rowptr[r0 + 1] - A.rowptr[r0]
    sel_ref = np.concatenate([np.arange(ref.rowptr[i], ref.rowptr[i + 1]) for i in (rows[0], rows[-1])])
    lo_r, hi_r = ref.rowptr[rows[0]], ref.rowptr[rows[-1] + 1]
    lo_a, hi_a = A.rowptr[rows[0]], A.rowptr[rows[-1] + 1]
    assert hi_r - lo_r == hi_a - lo_a and np.array_equal(ref.colidx[lo_r:hi_r], A.colidx[lo_a:hi_a])
    assert blockwise_rel_err(got[lo_a:hi_a], ref.vals[lo_r:hi_r], mag[lo_r:hi_r]) < TOL
    assert sel_ref.size > 0
    assert torch.equal(vals, plan.set_values(bsr.fem_q1_blocks(3, ne, 0, g.nelements, dev(g.element_data()[1].reshape(-1)),
                                                               dev(g.element_data()[0]), True)))


# ------------------------------------------------------------------ f4: second workload (Q2 rows, greedy aggregates)
def _second_workload(kind, small):
    if kind == "q2":
        g = pr.Generator(3, 6, seed=5, order=2) if small else pr.make_generator(5)
    else:
        g = pr.Generator(3, 14, seed=6, agg_mode=1) if small else pr.make_generator(6)
    g.build_prolongator(0)
    return g


@pytest.mark.parametrize("kind,small", [("q2", True), ("greedy", True), ("q2", False), ("greedy", False)])
def test_second_workload_hot_path(bsr, kind, small):
    """SpMV family (every entry), PtAP (structure ==, every block of AP and A_c against the oracle's form 2, a sample
    of coarse rows against the long-double form 1) and prolongator smoothing on the denser (Q2, up to 125 blocks per
    row, A_c rows of 125) and the irregular (greedy aggregates, A_c rows beyond 32 blocks) operators: output rows of
    more than 32 blocks run the staged kernels window by window; stage 1 of the Q2 operator, whose single rows exceed
    a brick's shared memory, runs the gather kernel."""
    from tests.test_gpu_fullsize import check_all_blocks, check_ptap_rows, check_spmv_family, sample_rows
    g = _second_workload(kind, small)
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    check_spmv_family(bsr, GA, GP, A, P, g.seed)
    plan = bsr.PtapPlan(GA, GP)
    (rap, cap), st = orc.ptap_symbolic(A, P)
    assert np.array_equal(plan.rowptr_c.cpu().numpy(), st[0]) and np.array_equal(plan.colidx_c.cpu().numpy(), st[1])
    rap_g, cap_g, _ = plan.ap_host()
    assert np.array_equal(rap_g, rap) and np.array_equal(cap_g, cap)
    sched = plan.schedule()
    if not small:
        assert np.diff(st[0]).max() > 32 and sched[2]["staged"]              # rows of several 32-slot windows, staged
        if kind == "q2":                                                    # one row of A with its P rows exceeds a brick
            assert (A.nbrows, A.nbrows * 3, A.nnzb) == (274625, 823875, 16974593) and not sched[1]["staged"]
        else:
            assert sched[1]["staged"]
    vals = plan.numeric()
    check_all_blocks(plan, vals, A, P, st, f"f4 {kind}")
    check_ptap_rows(plan, vals, A, P, st, sample_rows(P.nbcols, 8 if not small else 4, 11))
    import torch
    assert torch.equal(vals, plan.numeric())
    # prolongator smoothing on the same operator (P rows of up to 27 blocks for Q2)
    sm, _, _, pv, ref = smooth_check(bsr, A, g.P_tent(0), g.level_info(0)["omega"])
    assert np.abs(pv.cpu().numpy().reshape(ref.vals.shape) - P.vals).max() < 1e-13


# ------------------------------------------------------------------ f3: row sharding (library kernels per slab)
@pytest.mark.parametrize("d,ne,world", [(3, 11, 2), (3, 20, 3), (2, 62, 4)])
def test_row_sharded_hot_path_on_device(bsr, d, ne, world):
    """The sharded path of paper_2606_24748_b200/shard.py with the LIBRARY as the local kernel provider (bsr_spmv,
    bsr_gather_blocks, bsr_scatter_add_blocks, ptap_numeric, bcoo_set_values): `world` slabs of one problem driven by
    one host thread each on this GPU, exchanging through host queues (no kernel waits on another; the NCCL
    communicator of the multi-GPU launch is covered by the gloo test on the CPU).  Every slab must reproduce its rows
    of the single-rank oracle results."""
    import torch
    from paper_2606_24748_b200 import shard
    from tests.shard_util import LoopbackWorld, check_shard
    g = pr.Generator(d, ne, seed=2, modulus_mode=1)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    agg = g.level_arrays(0)["agg"].copy()
    x = pr.uniform(2, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
    xc = pr.uniform(2, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
    Ac = orc.ptap(A, P)
    dev0 = torch.device("cuda", 0)

    def rank(comm):
        torch.cuda.set_device(0)
        return check_shard(comm, shard.LibOps(dev0), A, P, agg, x, xc, Ac, to_dev=lambda t: t.to(dev0))

    res = LoopbackWorld(world).run(rank)
    for r in res:
        assert r["structure"], r
        assert max(r["spmv_A"], r["spmv_P"], r["spmv_Pt"], r["ptap"], r["ptap_scaled"]) < 1e-12, r
        assert r["gate_idle"] == 0 and r["gate_moved"] == 1, r
