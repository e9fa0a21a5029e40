"""Pins of the seeded input generator against what the paper and the mathematics fix."""
import numpy as np
import pytest

from paper_2606_24748_b200 import problems as pr

LAM = 0.3 / (1.3 * 0.4)
MU = 1 / (2 * 1.3)


def test_element_matrix_closed_forms():
    # I1: K_e[0][0] = (lambda + 3 mu)/3 in 2D, h (lambda + 4 mu)/9 in 3D; symmetric; rigid-body null space
    K2 = pr.element_matrix(2, 0.37)
    assert K2[0, 0] == pytest.approx((LAM + 3 * MU) / 3, rel=1e-14)
    h = 1 / 8
    K3 = pr.element_matrix(3, h)
    assert K3[0, 0] == pytest.approx(h * (LAM + 4 * MU) / 9, rel=1e-14)
    for K, nzero in ((K2, 3), (K3, 6)):
        assert np.abs(K - K.T).max() < 1e-16
        assert np.allclose(np.diag(K), K[0, 0], rtol=1e-13)
        w = np.linalg.eigvalsh(K)
        assert (np.abs(w) < 1e-13).sum() == nzero and w.min() > -1e-13


def test_golden_element_values():
    # tests/golden/element_matrix.txt: closed-form values from SURVEY.md I1 (E=1, nu=0.3)
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "element_matrix.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    assert pr.element_matrix(2, 1.0)[0, 0] == pytest.approx(vals["K2D_00"], rel=1e-13)
    assert pr.element_matrix(3, 1 / 8)[0, 0] == pytest.approx(vals["K3D_00_h8"], rel=1e-13)
    assert np.trace(pr.element_matrix(2, 1.0)) == pytest.approx(vals["trace2D"], rel=1e-5)
    assert np.trace(pr.element_matrix(3, 1 / 8)) == pytest.approx(vals["trace3D_h8"], rel=1e-5)


def rigid_modes(coords, d):
    n = coords.shape[0]
    nb = 6 if d == 3 else 3
    B = np.zeros((n, d, nb))
    for k in range(d):
        B[:, k, k] = 1
    x = coords
    if d == 3:
        B[:, 1, 3], B[:, 2, 3] = -x[:, 2], x[:, 1]      # e_0 x r
        B[:, 0, 4], B[:, 2, 4] = x[:, 2], -x[:, 0]      # e_1 x r
        B[:, 0, 5], B[:, 1, 5] = -x[:, 1], x[:, 0]      # e_2 x r
    else:
        B[:, 0, 2], B[:, 1, 2] = -x[:, 1], x[:, 0]
    return B.reshape(n * d, nb)


@pytest.mark.parametrize("d,ne", [(3, 6), (2, 9)])
def test_neumann_operator_annihilates_rigid_modes(d, ne):
    # I2 (rigid-body modes are the near-null space)
    g = pr.Generator(d, ne, seed=5, dirichlet=False)
    A = g.A(0)
    B = rigid_modes(g.level_arrays(0)["coords"], d)
    Ad = A.to_dense()
    assert np.abs(Ad @ B).max() < 1e-14 * max(1.0, np.abs(Ad).max()) * 10
    assert np.abs(Ad - Ad.T).max() < 1e-16


def test_dirichlet_operator_interior_rows(cfg0):
    # I2: with the clamped face, rows of nodes with ix >= 2 still annihilate the modes; A is SPD
    A = cfg0.A(0)
    n = 9
    B = rigid_modes(cfg0.level_arrays(0)["coords"], 3)
    Y = (A.to_scipy() @ B).reshape(-1, 3, 6)
    ix = np.arange(A.nbrows) % n
    assert np.abs(Y[ix >= 2]).max() < 1e-15
    Ad = A.to_dense()
    assert np.abs(Ad - Ad.T).max() < 1e-16
    assert np.linalg.eigvalsh(Ad).min() > 0


@pytest.mark.parametrize("d,ne", [(3, 8), (2, 8), (3, 5), (2, 512)])
def test_structure_counts(d, ne):
    # I3: nnzb(A) = (3n-2)^d for the clipped 3^d-point stencil; ascending columns
    g = pr.Generator(d, ne, seed=1)
    A = g.A(0)
    n = ne + 1
    assert A.nnzb == (3 * n - 2) ** d
    assert A.rowptr[0] == 0 and A.rowptr[-1] == A.nnzb
    i = 3 if ne < 100 else 1000
    row = A.colidx[A.rowptr[i]:A.rowptr[i + 1]]
    assert (np.diff(row) > 0).all()


def test_nnz_per_row_matches_paper():
    # PAPER.md:210-217 (Table 4): the Q1 operator has ~76 scalar nonzeros per row at the 1-GPU size (32^3 node
    # grid): counted on the generated matrix itself
    A = pr.Generator(3, 31, seed=1).A(0)
    assert A.nbrows == 32 ** 3
    assert 9 * A.nnzb / (3 * A.nbrows) == pytest.approx(76.0, abs=0.1)


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_tentative_prolongator(fix, request):
    # I4: P_tent^T P_tent = I.  I5: P_tent B_coarse = B_fine (modes reproduced exactly)
    g = request.getfixturevalue(fix)
    d = g.d
    Pt = g.P_tent(0).to_dense()
    assert np.abs(Pt.T @ Pt - np.eye(Pt.shape[1])).max() < 1e-14
    c1 = g.level_arrays(1)
    nb = 6 if d == 3 else 3
    # coarse modes about the origin: B_c(J) = R_J M(c_J - 0)
    Bf = rigid_modes(g.level_arrays(0)["coords"], d)
    Bc = np.zeros((Pt.shape[1], nb))
    for J in range(c1["coords"].shape[0]):
        M = rigid_modes(c1["coords"][J:J + 1], d)          # [I | W(c_J)] : d x nb
        Mfull = np.eye(nb)
        Mfull[:d, :] = M
        Bc[J * nb:(J + 1) * nb] = c1["rfac"][J] @ Mfull
    assert np.abs(Pt @ Bc - Bf).max() < 1e-14


def test_smoothed_prolongator_definition(cfg0):
    # O7: P = (I - omega D^-1 A) P_tent, dense check; omega = 4/(3 lambda); pattern = boolean A*P_tent
    A, Pt, P = cfg0.A(0).to_dense(), cfg0.P_tent(0).to_dense(), cfg0.P(0)
    info = cfg0.level_info(0)
    assert info["omega"] == pytest.approx(4 / (3 * info["lam"]), rel=1e-15)
    D = np.zeros_like(A)
    for i in range(0, A.shape[0], 3):
        D[i:i + 3, i:i + 3] = A[i:i + 3, i:i + 3]
    ref = Pt - info["omega"] * np.linalg.solve(D, A @ Pt)
    assert np.abs(P.to_dense() - ref).max() < 1e-14
    # lambda: 20 power iterations from the seeded start vector (R10)
    v = pr.uniform(0, pr.PURPOSE_POWER, A.shape[0])
    v /= np.linalg.norm(v)
    for _ in range(20):
        w = np.linalg.solve(D, A @ v)
        lam = np.linalg.norm(w)
        v = w / lam
    assert info["lam"] == pytest.approx(lam, rel=1e-12)
    assert P.nnzb == 2197  # SURVEY master table, config 0


def test_aggregate_counts():
    # O5 / R6 (merge rule): na = floor(n/3) boxes per side, the remainder merged into the last box
    for ne, na in ((8, 3), (10, 3), (12, 4)):      # n = ne+1 nodes per side -> floor(n/3) boxes per side
        gg = pr.Generator(3, ne, seed=0)
        gg.build_prolongator(0)
        assert gg.level_info(1)["nnodes"] == na ** 3 and gg.P(0).nbcols == na ** 3
    g = pr.Generator(3, 7, seed=0)   # 8 nodes per side: boxes of 3 and 5
    g.build_prolongator(0)
    agg = g.level_arrays(0)["agg"]
    assert agg.max() + 1 == 8
    sizes = np.bincount(agg)
    assert sorted(set(sizes.tolist())) == [27, 45, 75, 125]


def test_uniform_stream_reproducible():
    a = pr.uniform(3, pr.PURPOSE_FINE, 1000)
    b = pr.uniform(3, pr.PURPOSE_FINE, 1000)
    c = pr.uniform(3, pr.PURPOSE_COARSE, 1000)
    assert (a == b).all() and not (a == c).any()
    assert a.min() >= -1 and a.max() < 1 and abs(a.mean()) < 0.1


# ---------------------------------------------------------------- level 2 (O9, readings R9, R20; pin I5 second half)
def _coarse_modes(coords, rfac, d):
    nb = 6 if d == 3 else 3
    B = np.zeros((coords.shape[0] * nb, nb))
    for J in range(coords.shape[0]):
        Mfull = np.eye(nb)
        Mfull[:d, :] = rigid_modes(coords[J:J + 1], d)     # M(c_J - 0) = [[I, W(c_J)], [0, I]]
        B[J * nb:(J + 1) * nb] = rfac[J] @ Mfull
    return B


@pytest.mark.parametrize("d,ne", [(3, 17), (2, 26)])
def test_level2_tentative_prolongator(d, ne):
    """The level-2 tentative prolongator (6x6 / 3x3 blocks from the restricted rigid-body modes): orthonormal
    columns, and the fine rigid-body modes are reproduced through BOTH levels: P1_tent P2_tent B_2 = B_0."""
    from oracle import oracle as orc
    g = pr.Generator(d, ne, seed=9)
    g.build_prolongator(0)
    A0, P0 = g.A(0), g.P(0)
    Ac = orc.ptap(A0, P0)
    g.set_operator(1, pr.HostBSR(Ac.nbrows, Ac.nbcols, Ac.bs_r, Ac.bs_c, Ac.rowptr, Ac.colidx, Ac.vals))
    g.build_prolongator(1)
    nb = 6 if d == 3 else 3
    Pt1, Pt2 = g.P_tent(0).to_scipy().tocsr(), g.P_tent(1)
    assert (Pt2.bs_r, Pt2.bs_c) == (nb, nb) and Pt2.nbcols == g.level_info(2)["nnodes"] > 1
    Pt2 = Pt2.to_dense()
    assert np.abs(Pt2.T @ Pt2 - np.eye(Pt2.shape[1])).max() < 1e-14
    c1, c2 = g.level_arrays(1), g.level_arrays(2)
    B0 = rigid_modes(g.level_arrays(0)["coords"], d)
    B1 = _coarse_modes(c1["coords"], c1["rfac"], d)
    B2 = _coarse_modes(c2["coords"], c2["rfac"], d)
    assert np.abs(Pt2 @ B2 - B1).max() < 1e-13 * max(1.0, np.abs(B1).max())
    assert np.abs(Pt1 @ (Pt2 @ B2) - B0).max() < 1e-13
    # level-2 centroids are the unweighted means of their members' level-1 centroids (R20)
    agg = c1["agg"]
    for K in range(c2["coords"].shape[0]):
        assert np.allclose(c2["coords"][K], c1["coords"][agg == K].mean(axis=0), rtol=0, atol=1e-15)
    # smoothed level-2 prolongator against the dense formula with the 6x6 (3x3) block diagonal (O7 on A_1)
    A1 = g.A(1).to_dense()
    info = g.level_info(1)
    D = np.zeros_like(A1)
    for i in range(0, A1.shape[0], nb):
        D[i:i + nb, i:i + nb] = A1[i:i + nb, i:i + nb]
    ref = Pt2 - info["omega"] * np.linalg.solve(D, A1 @ Pt2)
    assert np.abs(g.P(1).to_dense() - ref).max() < 1e-13 * np.abs(ref).max()
    assert info["omega"] == pytest.approx(4 / (3 * info["lam"]), rel=1e-15)
