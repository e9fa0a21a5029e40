"""GPU parity of the V-cycle path (config 4's protocol O11 at a size the oracle does in
seconds): smoother, three-level V(2,2)-cycle with the dense coarsest solve, hierarchy recompute + refresh, 20 PCG
iterations.  Tolerances: V-cycle / smoother output 1e-10 relative in the 2-norm (a chain of ~20 SpMVs, each 1e-15
blockwise, through a preconditioner whose action has condition ~1e2); residual history 1e-8 (reading R18)."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr
from tests.util import blockwise_rel_err

pytestmark = pytest.mark.gpu


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


def as_host(M):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, M.vals)


@pytest.fixture(scope="module")
def three_level():
    """3D, 18^3 elements (19 nodes per side): 216 aggregates (bs 3 -> 6), then 8 (bs 6 -> 6), coarsest 48 dense."""
    g = pr.Generator(3, 18, seed=4)
    g.build_prolongator(0)
    A0, P0 = g.A(0), g.P(0)
    A1 = as_host(orc.ptap(A0, P0))
    g.set_operator(1, A1)
    g.build_prolongator(1)
    P1 = g.P(1)
    A2 = as_host(orc.ptap(A1, P1))
    lams = [g.level_info(0)["lam"], g.level_info(1)["lam"]]
    return g, [A0, A1, A2], [P0, P1], lams


def relerr(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_smoother_and_two_level(bsr):
    g = pr.make_generator(0)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = as_host(orc.ptap(A, P))
    lam = g.level_info(0)["lam"]
    H = orc.Hierarchy([A, Ac], [P], [lam])
    GA, GP, GAc = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P), bsr.Bsr.from_host(Ac)
    vc = bsr.VCycle([GA, GAc], [GP], [lam])
    n = A.nbrows * 3
    b = pr.uniform(0, pr.PURPOSE_RHS, n)
    x0 = pr.uniform(0, pr.PURPOSE_FINE, n)
    xs = vc.smooth(0, dev(b), dev(x0)).cpu().numpy()
    assert relerr(xs, H.smooth(0, b, x0)) < 1e-12
    z = vc.apply(dev(b)).cpu().numpy()
    assert relerr(z, H.vcycle(b)) < 1e-10
    # the V-cycle is a symmetric operator (pin I12), on the GPU too
    u = pr.uniform(0, pr.PURPOSE_FINE, n)
    zu = vc.apply(dev(u)).cpu().numpy()
    assert np.dot(u, z) == pytest.approx(np.dot(b, zu), rel=1e-9)


def test_three_level_vcycle_recompute_pcg(bsr, three_level):
    import torch
    g, As, Ps, lams = three_level
    A0, A1, A2 = As
    P0, P1 = Ps
    G0, GP0, GP1 = bsr.Bsr.from_host(A0), bsr.Bsr.from_host(P0), bsr.Bsr.from_host(P1)
    plan0 = bsr.PtapPlan(G0, GP0)
    assert np.array_equal(plan0.rowptr_c.cpu().numpy(), A1.rowptr) and np.array_equal(plan0.colidx_c.cpu().numpy(), A1.colidx)
    v1 = plan0.numeric()
    G1 = plan0.coarse_matrix(v1)
    plan1 = bsr.PtapPlan(G1, GP1)      # 6x6 * 6x6 products (<6,6,6>)
    assert np.array_equal(plan1.rowptr_c.cpu().numpy(), A2.rowptr) and np.array_equal(plan1.colidx_c.cpu().numpy(), A2.colidx)
    v2 = plan1.numeric()
    G2 = plan1.coarse_matrix(v2)
    a2 = v2.cpu().numpy().reshape(A2.vals.shape)
    scale = np.abs(A2.vals).max()
    assert np.abs(a2 - A2.vals).max() < 1e-12 * scale   # level-2 operator through two GPU products
    vc = bsr.VCycle([G0, G1, G2], [GP0, GP1], lams)
    H = orc.Hierarchy(As, Ps, lams)
    n = A0.nbrows * 3
    b = pr.uniform(4, pr.PURPOSE_RHS, n)
    db = dev(b)
    z = vc.apply(db).cpu().numpy()
    assert relerr(z, H.vcycle(b)) < 1e-10
    # level-1 smoother (6x6 blocks)
    b1 = pr.uniform(4, pr.PURPOSE_COARSE, A1.nbrows * 6)
    x1 = np.zeros_like(b1)
    assert relerr(vc.smooth(1, dev(b1), dev(x1)).cpu().numpy(), H.smooth(1, b1, x1)) < 1e-12
    # config 4's protocol: recompute the hierarchy (two ptap_numeric calls, level by level), refresh, 20 PCG iterations
    l0, a0 = bsr.counters()
    plan0.numeric(v1)
    G1.values_changed()
    plan1.numeric(v2)
    G2.values_changed()
    vc.refresh()
    x, hist = vc.pcg(db, 20)
    torch.cuda.synchronize()
    l1, a1 = bsr.counters()
    assert a1 == a0                         # no allocation in recompute, refresh, solve
    xo, ho = H.pcg(b, 20)
    hg = hist.cpu().numpy()
    assert np.abs(hg / ho - 1).max() < 1e-8, np.abs(hg / ho - 1).max()
    assert (np.diff(hg) < 0).all() and hg[-1] / hg[0] < 1e-6
    assert relerr(x.cpu().numpy(), xo) < 1e-8
    # determinism of the whole solve
    x2, hist2 = vc.pcg(db, 20)
    assert torch.equal(hist, hist2) and torch.equal(x, x2)


def test_vcycle_host_end_to_end(bsr):
    g = pr.make_generator(0)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = as_host(orc.ptap(A, P))
    lam = g.level_info(0)["lam"]
    vc = bsr.VCycle([bsr.Bsr.from_host(A), bsr.Bsr.from_host(Ac)], [bsr.Bsr.from_host(P)], [lam])
    b = pr.uniform(0, pr.PURPOSE_RHS, A.nbrows * 3)
    x = np.empty_like(b)
    vc.apply_host(b, x)
    assert relerr(x, orc.Hierarchy([A, Ac], [P], [lam]).vcycle(b)) < 1e-10


def test_vcycle_errors(bsr):
    g = pr.make_generator(0)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
    with pytest.raises(bsr.BsrError) as e:
        bsr.VCycle([GA, GA], [GP], [1.0])      # P does not connect A and A
    assert e.value.code == 2
    # a single level is a dense direct solve (2187 unknowns < 16384)
    one = bsr.VCycle([GA], [], [])
    b = pr.uniform(0, pr.PURPOSE_RHS, A.nbrows * 3)
    x = one.apply(dev(b)).cpu().numpy()
    assert relerr(orc.spmv(A, x), b) < 1e-9


@pytest.mark.parametrize("degree", [1, 3, 4])
def test_chebyshev_degrees(bsr, degree):
    """Degrees other than the default 2: degree 1 never forms a second residual, degrees >= 3 store r for the next
    step (from the zero guess only from step 1 on) and update it in place from step 2 on."""
    g = pr.make_generator(0)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = as_host(orc.ptap(A, P))
    lam = g.level_info(0)["lam"]
    H = orc.Hierarchy([A, Ac], [P], [lam], cheb_degree=degree)
    vc = bsr.VCycle([bsr.Bsr.from_host(A), bsr.Bsr.from_host(Ac)], [bsr.Bsr.from_host(P)], [lam], cheb_degree=degree)
    n = A.nbrows * 3
    b = pr.uniform(0, pr.PURPOSE_RHS, n)
    x0 = pr.uniform(0, pr.PURPOSE_FINE, n)
    assert relerr(vc.smooth(0, dev(b), dev(x0)).cpu().numpy(), H.smooth(0, b, x0)) < 1e-12
    assert relerr(vc.smooth(0, dev(b), dev(np.zeros(n))).cpu().numpy(), H.smooth(0, b, np.zeros(n))) < 1e-12
    assert relerr(vc.apply(dev(b)).cpu().numpy(), H.vcycle(b)) < 1e-10


def _dense(M):
    D = np.zeros((M.nbrows * M.bs_r, M.nbcols * M.bs_c))
    for i in range(M.nbrows):
        for k in range(M.rowptr[i], M.rowptr[i + 1]):
            j = M.colidx[k]
            D[i * M.bs_r:(i + 1) * M.bs_r, j * M.bs_c:(j + 1) * M.bs_c] = M.vals[k].reshape(M.bs_r, M.bs_c)
    return D


@pytest.mark.parametrize("case", ["tiny", "one_panel_and_a_bit", "banded", "not_banded"])
def test_coarsest_direct_solve(bsr, case):
    """The dense coarsest solve alone (a single level): x = L^-T (L^-1 b) against numpy's solve of the assembled matrix.
    Sizes below one 128-panel, just above one, several panels with a band, and the same operator under a random
    symmetric permutation of its block rows (no band: nothing is skipped)."""
    import scipy.sparse as sp
    if case == "tiny":
        g = pr.Generator(3, 2, seed=7)            # 27 nodes, 81 unknowns: one padded panel
        M = g.A(0)
    elif case == "one_panel_and_a_bit":
        g = pr.make_generator(0)
        g.build_prolongator(0)
        M = as_host(orc.ptap(g.A(0), g.P(0)))     # 27 aggregates x 6 = 162 unknowns, 6x6 blocks
    else:
        g = pr.Generator(3, 6, seed=7)            # 343 nodes, 1029 unknowns: 9 panels, half-bandwidth 57 nodes
        M = g.A(0)
        if case == "not_banded":
            S = sp.bsr_matrix((M.vals.reshape(-1, 3, 3), M.colidx, M.rowptr), shape=(M.nbrows * 3, M.nbrows * 3)).tocsr()
            perm = np.random.default_rng(3).permutation(M.nbrows)
            idx = (perm[:, None] * 3 + np.arange(3)[None, :]).ravel()
            S = S[idx][:, idx].tobsr(blocksize=(3, 3))
            S.sort_indices()
            M = pr.HostBSR(M.nbrows, M.nbrows, 3, 3, S.indptr.astype(np.int32), S.indices.astype(np.int32),
                           np.ascontiguousarray(S.data))
    D = _dense(M)
    assert np.allclose(D, D.T, rtol=1e-12, atol=1e-12 * np.abs(D).max())
    n = D.shape[0]
    b = pr.uniform(1, pr.PURPOSE_RHS, n)
    one = bsr.VCycle([bsr.Bsr.from_host(M)], [], [])
    x = one.apply(dev(b)).cpu().numpy()
    assert relerr(D @ x, b) < 1e-9
    assert relerr(x, np.linalg.solve(D, b)) < 1e-7
    one.refresh()                                  # a second factorisation into the same buffers
    assert np.array_equal(one.apply(dev(b)).cpu().numpy(), x)
