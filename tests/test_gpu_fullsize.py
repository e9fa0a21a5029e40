"""GPU parity at BASELINE.json's full sizes (configs 1-4), in the launch configuration bench.py times.

Structure is compared bit for bit over the whole matrix.  SpMV outputs are compared over every entry (the oracle's
long-double SpMV takes seconds).  EVERY block of AP and of A_c is compared with the oracle's form 2 (pinned to the
dense product in tests/test_oracle_pins.py; row-parallel, seconds at the full sizes), blockwise with the criterion
of tests/util.py, tolerance 1e-12 (north_star); the strict metric (plain ||O_b|| denominator) and the number of
blocks that needed the cancellation floor are printed.  A seeded sample of coarse rows is also compared with the
long-double form 1 (config 1: all rows).  Config 2 runs its ten-recompute protocol (reading R13, pin I9), every
recompute against the oracle's closed form; config 4 the three-level V-cycle / recompute / PCG protocol (O11) with the
residual-history tolerance 1e-8 (reading R18).  Where a product is chained (the coarse SpMV, A_2), the oracle is fed
the GPU's own intermediate so that the same 1e-12 bound applies."""
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


def absm(M):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, np.abs(M.vals))


def as_host(M, vals=None):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, M.vals if vals is None else vals)


def check_spmv_family(bsr, GA, GP, A, P, seed):
    x = pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
    xc = pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
    dx, dxc = dev(x), dev(xc)
    e = {}
    e["A"] = vec_blockwise_rel_err(GA.spmv(dx).cpu().numpy(), orc.spmv(A, x), A.bs_r, orc.spmv(absm(A), np.abs(x)))
    e["P"] = vec_blockwise_rel_err(GP.spmv(dxc).cpu().numpy(), orc.spmv(P, xc), P.bs_r, orc.spmv(absm(P), np.abs(xc)))
    e["Pt"] = vec_blockwise_rel_err(GP.spmv_t(dx).cpu().numpy(), orc.spmv_t(P, x), P.bs_c,
                                    orc.spmv_t(absm(P), np.abs(x)))
    assert max(e.values()) < TOL, e
    return e


def check_ptap_rows(plan, vals_c, A, P, structure, rows, scale=1.0):
    rc, cc = structure
    ref = orc.ptap(A, P, structure=structure, rows=rows)
    mag = orc.ptap(absm(A), absm(P), structure=structure, rows=rows)
    got = vals_c.cpu().numpy().reshape(-1, P.bs_c, P.bs_c)
    sel = np.concatenate([np.arange(rc[i], rc[i + 1]) for i in rows])
    err = blockwise_rel_err(got[sel], scale * ref.vals[sel], scale * mag.vals[sel])
    assert err < TOL, err
    return err


def strict_report(name, G, O, S, cfloor=1e-3):
    """The plain ||G_b - O_b|| / ||O_b|| metric over blocks with O_b != 0, and how many blocks the criterion of
    tests/util.py measured against the cancellation floor instead (reported, not asserted: R14)."""
    G, O, S = (np.asarray(t).reshape(O.shape[0], -1) for t in (G, O, S))
    on, sn = np.linalg.norm(O, axis=1), np.linalg.norm(S, axis=1)
    dn = np.linalg.norm(G - O, axis=1)
    nz = on > 0
    strict = float((dn[nz] / on[nz]).max()) if nz.any() else 0.0
    floored = int((on < cfloor * sn).sum())
    print(f"[parity] {name}: blocks {O.shape[0]}  strict max rel {strict:.2e}  floored blocks {floored}")
    return strict, floored


def check_all_blocks(plan, vals_c, A, P, structure, name, scale=1.0, f2=None, f2abs=None):
    """Every block of AP and A_c against the oracle's form 2 (all rows, element-wise criterion at 1e-12)."""
    if f2 is None:
        f2 = orc.PtapForm2(A, P)
        f2.run()
    if f2abs is None:
        f2abs = orc.PtapForm2(absm(A), absm(P))
        f2abs.run()
    assert np.array_equal(f2.rc, structure[0]) and np.array_equal(f2.cc, structure[1])
    _, _, ap = plan.ap_host()
    e_ap = blockwise_rel_err(ap, scale * f2.vals_ap, scale * f2abs.vals_ap)
    strict_report(name + " AP", ap, scale * f2.vals_ap, scale * f2abs.vals_ap)
    del ap
    got = vals_c.cpu().numpy().reshape(f2.vals_c.shape)
    e_c = blockwise_rel_err(got, scale * f2.vals_c, scale * f2abs.vals_c)
    strict_report(name + " A_c", got, scale * f2.vals_c, scale * f2abs.vals_c)
    assert e_ap < TOL and e_c < TOL, (e_ap, e_c)
    return f2, f2abs


def sample_rows(n, k, seed):
    rng = np.random.default_rng(seed)
    rows = np.unique(np.concatenate([[0, n - 1, n // 2], rng.choice(n, size=min(k, n), replace=False)]))
    return rows.astype(np.int32)


def setup(bsr, cfg):
    g = pr.make_generator(cfg)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    plan = bsr.PtapPlan(GA, GP)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    assert np.array_equal(plan.rowptr_c.cpu().numpy(), rc) and np.array_equal(plan.colidx_c.cpu().numpy(), cc)
    rap_g, cap_g, _ = plan.ap_host()
    assert np.array_equal(rap_g, rap) and np.array_equal(cap_g, cap)
    return g, A, P, GA, GP, plan, (rc, cc)


def test_config1_2d_all_small_shapes(bsr):
    """512^2 plane strain: 2x2, 2x3, 3x2 SpMV kernels, <2,2,3> and <3,2,3> products, 3x3 coarse operator."""
    g, A, P, GA, GP, plan, st = setup(bsr, 1)
    assert (A.nbrows, A.bs_r, P.bs_c, plan.nnzb_c) == (263169, 2, 3, 261121)      # SURVEY.md master table
    check_spmv_family(bsr, GA, GP, A, P, 1)
    vals = plan.numeric()
    check_ptap_rows(plan, vals, A, P, st, np.arange(P.nbcols, dtype=np.int32))
    check_all_blocks(plan, vals, A, P, st, "cfg1")
    # 3x3 SpMV on the coarse operator: the oracle multiplies the GPU's own A_c, so the 1e-12 bound applies
    Ac = pr.HostBSR(P.nbcols, P.nbcols, 3, 3, st[0], st[1], vals.cpu().numpy().reshape(-1, 3, 3))
    GAc = plan.coarse_matrix(vals)
    xc = pr.uniform(1, pr.PURPOSE_COARSE, Ac.nbrows * 3)
    assert vec_blockwise_rel_err(GAc.spmv(dev(xc)).cpu().numpy(), orc.spmv(Ac, xc), 3,
                                 orc.spmv(absm(Ac), np.abs(xc))) < TOL


def test_config2_recompute_protocol(bsr):
    """64^3: SpMV family, then ten numeric recomputes over one cached plan, A rescaled by s_k (R13)."""
    g, A, P, GA, GP, plan, st = setup(bsr, 2)
    assert (plan.nbrows_c, plan.nnzb_c) == (9261, 226981)
    check_spmv_family(bsr, GA, GP, A, P, 2)
    rows = sample_rows(P.nbcols, 48, 2)
    out = plan.new_values()
    plan.numeric(out)
    check_ptap_rows(plan, out, A, P, st, rows)
    f2, f2abs = check_all_blocks(plan, out, A, P, st, "cfg2")
    builds = plan.info()["n_r_value_builds"]
    s = pr.uniform(2, pr.PURPOSE_RESCALE, 10, 0.5, 2.0)
    a0 = bsr.counters()[1]
    ref0, mag0 = f2.vals_c, f2abs.vals_c                        # the ORACLE's A_c^(0) and its magnitude sum
    for k, sk in enumerate(s):
        GA.vals.copy_(dev(A.vals.reshape(-1)) * sk)
        GA.values_changed()
        plan.numeric(out)
        # every recompute, every block, against the oracle's closed form I9: A_c^(k) = s_k A_c^(0) (pinned for the
        # oracle in tests/test_oracle_pins.py::test_recompute_scaling_closed_form)
        got = out.cpu().numpy().reshape(ref0.shape)
        assert blockwise_rel_err(got, sk * ref0, sk * mag0) < TOL, k
    check_ptap_rows(plan, out, A, P, st, rows[:8], scale=float(s[-1]))
    check_all_blocks(plan, out, A, P, st, "cfg2 recompute 10", scale=float(s[-1]), f2=f2, f2abs=f2abs)
    assert bsr.counters()[1] == a0                              # no allocation in the hot recomputes
    assert plan.info()["n_r_value_builds"] == builds            # P untouched: the R cache was never rebuilt


def test_config3_headline_grid(bsr):
    """128^3, lognormal modulus: the grid bench.py times."""
    g, A, P, GA, GP, plan, st = setup(bsr, 3)
    assert (A.nbrows, A.nnzb, P.nnzb, plan.nnzb_c) == (2146689, 57066625, 9663597, 2048383)
    info = plan.info()
    assert (info["nnzb_ap"], info["n_products_1"], info["n_products_2"]) == (26198073, 258474853, 100544625)
    assert abs(info["algorithmic_bytes"] - 15.585e9) < 2e6
    check_spmv_family(bsr, GA, GP, A, P, 3)
    vals = plan.numeric()
    check_ptap_rows(plan, vals, A, P, st, sample_rows(P.nbcols, 40, 3))
    check_all_blocks(plan, vals, A, P, st, "cfg3")
    import torch
    assert torch.equal(vals, plan.numeric())                    # bit-reproducible


def test_config4_three_level_protocol(bsr):
    """96^3, three levels: V(2,2)-cycle, full hierarchy recompute, 20 PCG iterations (O11)."""
    import torch
    g, A0, P0, G0, GP0, plan0, st0 = setup(bsr, 4)
    v1 = plan0.numeric()
    check_ptap_rows(plan0, v1, A0, P0, st0, sample_rows(P0.nbcols, 24, 4))
    f2, _ = check_all_blocks(plan0, v1, A0, P0, st0, "cfg4 L0->L1")
    A1 = as_host(f2.run(), f2.vals_c.copy())
    assert (A1.nbrows, A1.nnzb) == (32768, 830584)
    g.set_operator(1, A1)
    g.build_prolongator(1)
    P1 = g.P(1)
    G1 = plan0.coarse_matrix(v1)                                # the GPU's own level-1 operator
    GP1 = bsr.Bsr.from_host(P1)
    plan1 = bsr.PtapPlan(G1, GP1)
    (_, _), st1 = orc.ptap_symbolic(A1, P1)
    assert np.array_equal(plan1.rowptr_c.cpu().numpy(), st1[0]) and np.array_equal(plan1.colidx_c.cpu().numpy(), st1[1])
    v2 = plan1.numeric()
    # chained product: the oracle multiplies the GPU's own A_1 (same structure), so the 1e-12 bound applies to A_2
    A1g = as_host(A1, v1.cpu().numpy().reshape(A1.vals.shape))
    check_all_blocks(plan1, v2, A1g, P1, st1, "cfg4 L1->L2")
    A2 = as_host(orc.ptap(A1g, P1, structure=st1))
    assert (A2.nbrows, A2.nnzb) == (1000, 21952)
    mag2 = orc.ptap(absm(A1g), absm(P1), structure=st1).vals
    assert blockwise_rel_err(v2.cpu().numpy().reshape(A2.vals.shape), A2.vals, mag2) < TOL
    G2 = plan1.coarse_matrix(v2)
    lams = [g.level_info(0)["lam"], g.level_info(1)["lam"]]
    vc = bsr.VCycle([G0, G1, G2], [GP0, GP1], lams)
    H = orc.Hierarchy([A0, A1, A2], [P0, P1], lams)
    b = pr.uniform(4, pr.PURPOSE_RHS, A0.nbrows * 3)
    db = dev(b)
    z, zo = vc.apply(db).cpu().numpy(), H.vcycle(b)
    assert np.linalg.norm(z - zo) < 1e-9 * np.linalg.norm(zo)
    plan0.numeric(v1); G1.values_changed()
    plan1.numeric(v2); G2.values_changed()
    vc.refresh()
    x, hist = vc.pcg(db, 20)
    xo, ho = H.pcg(b, 20)
    hg = hist.cpu().numpy()
    assert np.abs(hg / ho - 1).max() < 1e-8, np.abs(hg / ho - 1).max()
    assert (np.diff(hg) < 0).all()
