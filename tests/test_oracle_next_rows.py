"""Pins of the oracle routines behind SURVEY.md 8(f) rows f1 (prolongator smoothing) and f2 (blocked COO assembly)
against what the paper and the mathematics fix -- dense formulas through numpy's own solver, scipy's coordinate-format
duplicate summation, exact mode reproduction, special cases -- and against the generator's independent host assembly.
All `-m "not gpu"`."""
import numpy as np
import pytest
import scipy.sparse as sp

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr
from tests.test_generator import _coarse_modes, rigid_modes


def _dense_smoothed(A, Pt, bs, omega):
    """PAPER.md:54-56 written densely: P = P~ - omega D^-1 (A P~), D the bs x bs block diagonal (R11)."""
    D = np.zeros_like(A)
    for i in range(0, A.shape[0], bs):
        D[i:i + bs, i:i + bs] = A[i:i + bs, i:i + bs]
    return Pt - omega * np.linalg.solve(D, A @ Pt)


# ------------------------------------------------------------------ f1: prolongator smoothing
@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_prolongator_smooth_vs_dense_formula(fix, request):
    g = request.getfixturevalue(fix)
    A, Pt = g.A(0), g.P_tent(0)
    for omega in (g.level_info(0)["omega"], 0.0, -0.73):
        P = orc.prolongator_smooth(A, Pt, omega)
        ref = _dense_smoothed(A.to_dense(), Pt.to_dense(), A.bs_r, omega)
        got = pr.HostBSR(P.nbrows, P.nbcols, P.bs_r, P.bs_c, P.rowptr, P.colidx, P.vals).to_dense()
        assert np.abs(got - ref).max() < 1e-14 * max(1.0, np.abs(ref).max())
    # omega = 0: P is P~ on the larger pattern (the block AXPY adds P~ on a subset of the pattern)
    P0 = orc.prolongator_smooth(A, Pt, 0.0)
    assert np.count_nonzero(np.abs(P0.vals).reshape(P0.nnzb, -1).max(axis=1)) == Pt.nnzb
    # pattern = boolean pattern of A * P~ (R5), from a library boolean product
    S = (sp.csr_matrix((np.ones(A.nnzb), A.colidx, A.rowptr), shape=(A.nbrows, A.nbcols)) @
         sp.csr_matrix((np.ones(Pt.nnzb), Pt.colidx, Pt.rowptr), shape=(Pt.nbrows, Pt.nbcols))).tocsr()
    S.sort_indices()
    assert np.array_equal(S.indptr, P0.rowptr) and np.array_equal(S.indices, P0.colidx)


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_prolongator_smooth_matches_generator(fix, request):
    """The generator's own host loop (an independent implementation) gives the same P."""
    g = request.getfixturevalue(fix)
    P, Pg = orc.prolongator_smooth(g.A(0), g.P_tent(0), g.level_info(0)["omega"]), g.P(0)
    assert np.array_equal(P.rowptr, Pg.rowptr) and np.array_equal(P.colidx, Pg.colidx)
    assert np.abs(P.vals - Pg.vals).max() < 1e-15


@pytest.mark.parametrize("d,ne", [(3, 6), (2, 9)])
def test_smoothed_prolongator_reproduces_rigid_modes_on_neumann_problem(d, ne):
    """A B_0 = 0 on a Neumann problem, so (I - omega D^-1 A) keeps the exact reproduction P B_c = B_0 of the
    tentative prolongator (the near-null space is represented exactly on the coarse level)."""
    g = pr.Generator(d, ne, seed=5, dirichlet=False)
    g.build_prolongator(0)
    P = orc.prolongator_smooth(g.A(0), g.P_tent(0), 0.61)
    Pd = pr.HostBSR(P.nbrows, P.nbcols, P.bs_r, P.bs_c, P.rowptr, P.colidx, P.vals).to_dense()
    B0 = rigid_modes(g.level_arrays(0)["coords"], d)
    c1 = g.level_arrays(1)
    Bc = _coarse_modes(c1["coords"], c1["rfac"], d)
    assert np.abs(Pd @ Bc - B0).max() < 1e-13


def test_prolongator_smooth_level2_six_by_six_blocks():
    """The 6x6 case (level 1 -> level 2 of config 4's recipe): dense formula with numpy's solve on the 6x6 blocks."""
    g = pr.Generator(3, 8, seed=11)
    g.build_prolongator(0)
    Ac = orc.ptap(g.A(0), g.P(0))
    A1 = pr.HostBSR(Ac.nbrows, Ac.nbcols, 6, 6, Ac.rowptr, Ac.colidx, Ac.vals)
    g.set_operator(1, A1)
    g.build_prolongator(1)
    Pt = g.P_tent(1)
    om = g.level_info(1)["omega"]
    P = orc.prolongator_smooth(A1, Pt, om)
    ref = _dense_smoothed(A1.to_dense(), Pt.to_dense(), 6, om)
    got = pr.HostBSR(P.nbrows, P.nbcols, 6, 6, P.rowptr, P.colidx, P.vals).to_dense()
    assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max()
    assert np.abs(P.vals - g.P(1).vals).max() < 1e-14


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_power_lambda(fix, request):
    """R10: 20 power iterations on D^-1 A from the seeded start vector -- against the generator's own loop, a dense
    numpy iteration through numpy's solver, and the bound by the true spectral radius (scipy eigenvalues)."""
    g = request.getfixturevalue(fix)
    A = g.A(0)
    n, bs = A.nbrows * A.bs_r, A.bs_r
    v0 = pr.uniform(g.seed, pr.PURPOSE_POWER, n)
    lam = orc.power_lambda(A, v0, 20)
    assert lam == pytest.approx(g.level_info(0)["lam"], rel=1e-13)
    Ad = A.to_dense()
    D = np.zeros_like(Ad)
    for i in range(0, n, bs):
        D[i:i + bs, i:i + bs] = Ad[i:i + bs, i:i + bs]
    v = v0 / np.linalg.norm(v0)
    for _ in range(20):
        w = np.linalg.solve(D, Ad @ v)
        ref = np.linalg.norm(w)
        v = w / ref
    assert lam == pytest.approx(ref, rel=1e-12)
    rho = np.abs(np.linalg.eigvals(np.linalg.solve(D, Ad))).max()
    assert 0.8 * rho < lam <= rho * (1 + 1e-12)            # a lower estimate of the spectral radius (D^-1 A ~ SPD)
    assert orc.power_lambda(A, 3.7 * v0, 20) == pytest.approx(lam, rel=1e-14)    # the start vector is normalised
    assert orc.power_lambda(A, v0, 1) != pytest.approx(lam, rel=1e-6)            # and the iteration count matters


def test_prolongator_smooth_rejects_missing_diagonal():
    A = pr.HostBSR(2, 2, 2, 2, np.array([0, 1, 2], np.int32), np.array([1, 0], np.int32), np.ones((2, 2, 2)))
    Pt = pr.HostBSR(2, 1, 2, 3, np.array([0, 1, 2], np.int32), np.array([0, 0], np.int32), np.ones((2, 2, 3)))
    with pytest.raises(RuntimeError):
        orc.prolongator_smooth(A, Pt, 0.5)


# ------------------------------------------------------------------ f2: blocked COO assembly
def _scalar_coo(brow, bcol, stream, nbrows, nbcols):
    """The same stream as SCALAR coordinates, summed by scipy's COO -> CSR conversion (duplicates are added)."""
    n, br, bc = stream.shape
    r = (brow[:, None, None] * br + np.arange(br)[None, :, None] + np.zeros((1, 1, bc), int)).ravel()
    c = (bcol[:, None, None] * bc + np.arange(bc)[None, None, :] + np.zeros((1, br, 1), int)).ravel()
    return sp.coo_matrix((stream.ravel(), (r, c)), shape=(nbrows * br, nbcols * bc)).tocsr()


@pytest.mark.parametrize("br,bc", [(3, 3), (2, 3), (3, 6), (6, 6)])
def test_bcoo_vs_scipy_duplicate_summation(br, bc):
    rng = np.random.default_rng(br * 10 + bc)
    nbrows, nbcols, n = 37, 29, 900
    brow = rng.integers(0, nbrows, n).astype(np.int32)
    bcol = rng.integers(0, nbcols, n).astype(np.int32)
    brow[:40] = 5                                        # a heavily duplicated row; row 7 stays empty
    bcol[:40] = rng.integers(0, 3, 40)
    keep = brow != 7
    brow, bcol = brow[keep], bcol[keep]
    stream = rng.uniform(-1, 1, (brow.shape[0], br, bc))
    M = orc.bcoo_assemble(brow, bcol, stream, nbrows, nbcols)
    # structure: one block per distinct coordinate, rows in order, columns strictly ascending
    key = np.unique(brow.astype(np.int64) * nbcols + bcol)
    assert M.nnzb == key.shape[0] and M.rowptr[8] == M.rowptr[7]
    assert np.array_equal(M.colidx, (key % nbcols).astype(np.int32))
    assert np.array_equal(np.diff(M.rowptr), np.bincount((key // nbcols).astype(int), minlength=nbrows))
    got = pr.HostBSR(nbrows, nbcols, br, bc, M.rowptr, M.colidx, M.vals).to_dense()
    ref = np.asarray(_scalar_coo(brow, bcol, stream, nbrows, nbcols).todense())
    assert np.abs(got - ref).max() < 1e-14
    # brute force: dense scatter-add in declaration order
    D = np.zeros((nbrows * br, nbcols * bc))
    for c in range(brow.shape[0]):
        D[brow[c] * br:(brow[c] + 1) * br, bcol[c] * bc:(bcol[c] + 1) * bc] += stream[c]
    assert np.abs(got - D).max() < 1e-14


def test_bcoo_without_duplicates_is_a_permutation():
    rng = np.random.default_rng(3)
    nbrows = nbcols = 11
    key = rng.permutation(nbrows * nbcols)[:60]
    brow, bcol = (key // nbcols).astype(np.int32), (key % nbcols).astype(np.int32)
    stream = rng.uniform(-1, 1, (60, 3, 6))
    M = orc.bcoo_assemble(brow, bcol, stream, nbrows, nbcols)
    order = np.argsort(key, kind="stable")
    assert np.array_equal(M.vals, stream[order])          # bit for bit: nothing is added


def test_bcoo_negative_coordinates_are_ignored():
    rng = np.random.default_rng(8)
    n, nb = 400, 13
    brow, bcol = rng.integers(0, nb, n).astype(np.int32), rng.integers(0, nb, n).astype(np.int32)
    stream = rng.uniform(-1, 1, (n, 2, 3))
    drop = rng.random(n) < 0.3
    b2, c2 = brow.copy(), bcol.copy()
    b2[drop & (np.arange(n) % 2 == 0)] = -1
    c2[drop & (np.arange(n) % 2 == 1)] = -7
    M = orc.bcoo_assemble(b2, c2, stream, nb, nb)
    ref = orc.bcoo_assemble(brow[~drop], bcol[~drop], stream[~drop], nb, nb)
    assert np.array_equal(M.rowptr, ref.rowptr) and np.array_equal(M.colidx, ref.colidx) and np.array_equal(M.vals, ref.vals)


def test_bcoo_rejects_bad_coordinates():
    with pytest.raises(RuntimeError):
        orc.bcoo_assemble(np.array([0, 4], np.int32), np.array([0, 0], np.int32), np.zeros((2, 2, 2)), 3, 3)
    M = orc.bcoo_assemble(np.array([0], np.int32), np.array([1], np.int32), np.ones((1, 2, 2)), 2, 2)
    with pytest.raises(RuntimeError):                      # a coordinate outside a given structure
        orc.bcoo_assemble(np.array([1], np.int32), np.array([1], np.int32), np.ones((1, 2, 2)), 2, 2,
                          structure=(M.rowptr, M.colidx))


@pytest.mark.parametrize("d,ne,mode,dirichlet", [(3, 8, 0, True), (3, 5, 1, True), (2, 9, 1, False), (2, 12, 0, True)])
def test_finite_element_stream_assembles_the_operator(d, ne, mode, dirichlet):
    """Finite-element assembly through the primitive: the element contribution stream of the
    generator, summed by the oracle, is the generator's own gather-form operator (structure ==, values to rounding),
    clamped face included."""
    g = pr.Generator(d, ne, seed=3, modulus_mode=mode, dirichlet=dirichlet)
    A = g.A(0)
    brow, bcol, blocks = g.element_stream()
    assert brow.shape[0] == ne ** d * 4 ** d
    M = orc.bcoo_assemble(brow, bcol, blocks, A.nbrows, A.nbcols)
    assert np.array_equal(M.rowptr, A.rowptr) and np.array_equal(M.colidx, A.colidx)
    assert np.abs(M.vals - A.vals).max() < 1e-14 * np.abs(A.vals).max()
    # contributions per block row: (elements adjacent to the node) x 2^d, from 2^d at a corner to 4^d inside
    seg = np.bincount(brow, minlength=A.nbrows)
    assert seg.max() == 4 ** d and seg.min() == 2 ** d
    # an element range gives the same coordinates as the matching slice of the full stream
    e0, e1 = 3, 7
    b2, c2, v2 = g.element_stream(e0, e1)
    s = slice(e0 * 4 ** d, e1 * 4 ** d)
    assert np.array_equal(b2, brow[s]) and np.array_equal(c2, bcol[s]) and np.array_equal(v2, blocks[s])
