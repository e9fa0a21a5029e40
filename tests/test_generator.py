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
    # PAPER.md:210-217 (Table 4): Q1 operator has ~76 nonzeros per row at the 1-GPU size (32^3 node grid)
    m = 32
    assert 3 * (3 * m - 2) ** 3 / m ** 3 == pytest.approx(76.0, abs=0.1)


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
    # O5 / R6 (merge rule): 27 aggregates at cfg0; 21^3 at 65^3 nodes; 32^3 at 97^3 nodes (counted without
    # building those grids: na = floor(n/3))
    assert (9 // 3) ** 3 == 27 and (65 // 3) ** 3 == 9261 and (97 // 3) ** 3 == 32768 and (129 // 3) ** 3 == 79507
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
