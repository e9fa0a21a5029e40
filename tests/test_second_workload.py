"""the second workload of the seeded generator -- Q2 elements (denser rows)
and greedy (MIS-like) aggregates -- pinned against what the mathematics fixes, and the oracle's
PtAP / the host plan of the CUDA library exercised off the regular 27-point happy path.  All `-m "not gpu"`."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import bsr, problems as pr
from tests.test_generator import LAM, MU, _coarse_modes, rigid_modes


def _as_host(M):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, M.vals)


@pytest.mark.parametrize("d", [2, 3])
def test_q2_element_matrix(d):
    h = 0.5
    K = pr.element_matrix(d, h, order=2)
    nen = 3 ** d
    assert K.shape == (d * nen, d * nen) and np.abs(K - K.T).max() < 1e-15
    w = np.linalg.eigvalsh(K)
    assert (np.abs(w) < 1e-13).sum() == (6 if d == 3 else 3) and w.min() > -1e-13
    # closed form: the quadratic field u = (x^2, 0[, 0]) is in the Q2 space; its strain energy on [0,h]^d is
    # 1/2 (lambda + 2 mu) int (2x)^2 = (lambda + 2 mu) * (2/3) h^3 * h^(d-1)   (plane strain in 2D)
    idx = np.arange(nen)
    xs = (idx % 3) * (h / 2)
    u = np.zeros(d * nen)
    u[0::d] = xs ** 2
    assert u @ K @ u == pytest.approx((LAM + 2 * MU) * (4.0 / 3.0) * h ** 3 * h ** (d - 1), rel=1e-13)
    # patch test: a linear field (constant strain) produces no force on the element's interior node
    lin = np.zeros(d * nen)
    ys = ((idx // 3) % 3) * (h / 2)
    lin[0::d] = 0.3 * xs + 0.1 * ys
    lin[1::d] = -0.2 * xs
    centre = (nen - 1) // 2
    assert np.abs((K @ lin)[d * centre:d * centre + d]).max() < 1e-14
    # the corner-only restriction of a Q2 element is not the Q1 element (a wrong order switch would pass otherwise)
    assert pr.element_matrix(d, h, order=1).shape == (d * 2 ** d, d * 2 ** d)


@pytest.mark.parametrize("d,ne", [(3, 4), (2, 7)])
def test_q2_operator_structure_and_null_space(d, ne):
    g = pr.Generator(d, ne, seed=2, order=2, dirichlet=False)
    A = g.A(0)
    n = 2 * ne + 1
    assert A.nbrows == n ** d
    # closed form: per direction, corner nodes couple to 5 (3 at the ends), mid nodes to 3 nodes
    per_dim = (ne - 1) * 5 + 2 * 3 + ne * 3
    assert A.nnzb == per_dim ** d
    for i in range(A.nbrows):
        c = A.colidx[A.rowptr[i]:A.rowptr[i + 1]]
        assert (np.diff(c) > 0).all()
    Ad = A.to_dense()
    assert np.abs(Ad - Ad.T).max() < 1e-14
    B = rigid_modes(g.level_arrays(0)["coords"], d)
    assert np.abs(Ad @ B).max() < 1e-13                       # rigid-body modes are the near-null space
    # finite-element stream of the same operator through the oracle's blocked COO assembly (3^(2d) per element)
    brow, bcol, blocks = g.element_stream()
    assert brow.shape[0] == ne ** d * 9 ** d
    M = orc.bcoo_assemble(brow, bcol, blocks, A.nbrows, A.nbcols)
    assert np.array_equal(M.rowptr, A.rowptr) and np.array_equal(M.colidx, A.colidx)
    assert np.abs(M.vals - A.vals).max() < 1e-14 * np.abs(A.vals).max()


def test_q2_nonzeros_per_row_near_the_papers():
    # PAPER.md:206-217, Table 4: the Q2 harness has 169 (n=1) to 180 (n=8) nonzeros per row, Q1 76-78
    g = pr.Generator(3, 16, seed=0, order=2)
    A = g.A(0)
    nnz_row = A.nnzb * 9 / (A.nbrows * 3)
    assert 165 < nnz_row < 195, nnz_row
    g = pr.Generator(3, 32, seed=0)
    A1 = g.A(0)
    assert A1.nbrows == A.nbrows and 2.2 < (A.nnzb / A1.nnzb) < 2.5     # same node grid, ~2.3x the blocks


@pytest.mark.parametrize("d,ne,order", [(3, 9, 1), (2, 20, 1), (3, 4, 2)])
def test_greedy_aggregates(d, ne, order):
    g = pr.Generator(d, ne, seed=6, agg_mode=1, order=order, dirichlet=False)
    g.build_prolongator(0)
    A, Pt, P = g.A(0), g.P_tent(0), g.P(0)
    agg = g.level_arrays(0)["agg"]
    na = P.nbcols
    sizes = np.bincount(agg, minlength=na)
    assert agg.min() == 0 and agg.max() == na - 1 and sizes.min() >= 4            # a disjoint cover, no tiny aggregate
    assert len(set(sizes.tolist())) > 3                                          # irregular sizes
    # every root aggregate holds a node together with ALL its neighbours (greedy covering)
    full = 0
    for J in range(na):
        mem = set(np.nonzero(agg == J)[0].tolist())
        full += any(set(A.colidx[A.rowptr[i]:A.rowptr[i + 1]].tolist()) <= mem for i in mem)
    assert full == na
    # orthonormal tentative blocks and exact mode reproduction, also through the smoothed P
    Ptd = Pt.to_dense()
    assert np.abs(Ptd.T @ Ptd - np.eye(Ptd.shape[1])).max() < 1e-13
    B0 = rigid_modes(g.level_arrays(0)["coords"], d)
    c1 = g.level_arrays(1)
    Bc = _coarse_modes(c1["coords"], c1["rfac"], d)
    assert np.abs(Ptd @ Bc - B0).max() < 1e-12
    assert np.abs(P.to_dense() @ Bc - B0).max() < 1e-12                            # Neumann problem: A B_0 = 0
    # same seed, same aggregates; another seed, others
    g2 = pr.Generator(d, ne, seed=6, agg_mode=1, order=order, dirichlet=False); g2.build_prolongator(0)
    g3 = pr.Generator(d, ne, seed=7, agg_mode=1, order=order, dirichlet=False); g3.build_prolongator(0)
    assert np.array_equal(agg, g2.level_arrays(0)["agg"]) and not np.array_equal(agg, g3.level_arrays(0)["agg"])
    # the oracle's prolongator smoothing reproduces the generator's P on the irregular pattern
    Po = orc.prolongator_smooth(A, Pt, g.level_info(0)["omega"])
    assert np.array_equal(Po.colidx, P.colidx) and np.abs(Po.vals - P.vals).max() < 1e-14


def test_row_lengths_beyond_one_window():
    """At sizes with an interior both variants have rows of more than 32 output blocks.  The staged PtAP schedule cuts
    such rows into windows of 32 slots (stage 2: one brick per window of a coarse row); it covers every block product
    exactly once.  Only stage 1 of the Q2 operator stays on the gather kernels: a single row of A (125 blocks) with the
    P rows it references (up to 27 blocks each) exceeds the shared memory of a brick."""
    g = pr.Generator(3, 12, seed=5, order=2); g.build_prolongator(0)
    hp = bsr.HostPlan(g.A(0), g.P(0))
    assert np.diff(hp.rowptr_ap).max() == 64 and np.diff(hp.rowptr_c).max() == 125 and np.diff(g.P(0).rowptr).max() == 27
    s1, s2 = hp.stream_stats[1], hp.stream_stats[2]
    assert s1["ok"] == 0
    assert s2["ok"] == 1 and s2["mask_bits"] == hp.t2.shape[0] and s2["max_smem"] <= 75000
    assert s2["bricks"] == int(np.sum((np.diff(hp.rowptr_c) + 31) // 32))           # one brick per window
    g = pr.Generator(3, 24, seed=6, agg_mode=1); g.build_prolongator(0)
    hp = bsr.HostPlan(g.A(0), g.P(0))
    assert np.diff(hp.rowptr_c).max() > 32
    s1, s2 = hp.stream_stats[1], hp.stream_stats[2]
    assert s1["ok"] == 1 and s1["mask_bits"] == hp.k1.shape[0]
    assert s2["ok"] == 1 and s2["mask_bits"] == hp.t2.shape[0]
    assert s2["bricks"] == int(np.sum(np.maximum(1, (np.diff(hp.rowptr_c) + 31) // 32)))


@pytest.mark.parametrize("kind", ["q2", "greedy"])
def test_ptap_off_the_regular_path(kind):
    """Oracle forms 1 and 2 against the dense triple product, and the CUDA library's host plan against the oracle's
    symbolic structure, on rows denser / more irregular than the 27-point box case."""
    g = pr.Generator(3, 3, seed=3, order=2) if kind == "q2" else pr.Generator(3, 8, seed=3, agg_mode=1)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = orc.ptap(A, P)
    dense = P.to_dense().T @ A.to_dense() @ P.to_dense()
    assert np.abs(_as_host(Ac).to_dense() - dense).max() < 1e-13 * np.abs(dense).max()
    f2 = orc.PtapForm2(A, P)
    assert np.abs(f2.run().vals - Ac.vals).max() < 1e-13 * np.abs(Ac.vals).max()
    hp = bsr.HostPlan(A, P)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    assert np.array_equal(hp.rowptr_ap, rap) and np.array_equal(hp.colidx_ap, cap)
    assert np.array_equal(hp.rowptr_c, rc) and np.array_equal(hp.colidx_c, cc)
    # every block product appears exactly once in the gather lists
    assert hp.k1.shape[0] == sum(P.rowptr[j + 1] - P.rowptr[j] for j in A.colidx)
    if kind == "q2":
        assert np.diff(A.rowptr).max() == 125                 # a corner node of the Q2 grid couples to 5^3 nodes
    else:
        assert len(set(np.diff(rc).tolist())) > 5 and len(set(np.diff(P.rowptr).tolist())) > 3   # irregular rows
