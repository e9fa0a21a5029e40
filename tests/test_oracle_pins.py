"""Pins of the CPU oracle against things other than itself:
dense brute force, scipy.sparse library routines, closed forms and invariants."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr
from tests.util import blockwise_rel_err, vec_blockwise_rel_err
from tests.test_generator import rigid_modes


def dense_blocks(M, rowptr, colidx, br, bc):
    out = np.empty((colidx.shape[0], br, bc))
    for i in range(rowptr.shape[0] - 1):
        for k in range(rowptr[i], rowptr[i + 1]):
            j = colidx[k]
            out[k] = M[i * br:(i + 1) * br, j * bc:(j + 1) * bc]
    return out


# ---------------------------------------------------------------- SpMV family (I10)
@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_spmv_family_vs_dense(fix, request):
    g = request.getfixturevalue(fix)
    A, P = g.A(0), g.P(0)
    x = pr.uniform(g.seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
    xc = pr.uniform(g.seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
    Ad, Pd = A.to_dense(), P.to_dense()
    assert vec_blockwise_rel_err(orc.spmv(A, x), Ad @ x, A.bs_r) < 1e-13
    assert vec_blockwise_rel_err(orc.spmv(P, xc), Pd @ xc, P.bs_r) < 1e-13
    assert vec_blockwise_rel_err(orc.spmv_t(P, x), Pd.T @ x, P.bs_c) < 1e-13
    assert vec_blockwise_rel_err(orc.spmv_fast(A, x), Ad @ x, A.bs_r) < 1e-13


def test_spmv_bsr_vs_scalar_csr_library():
    # blocked and scalar formats give the same answers -> scipy CSR expansion, config-1-like 2D
    g = pr.Generator(2, 40, seed=1)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    x = pr.uniform(1, pr.PURPOSE_FINE, A.nbrows * 2)
    xc = pr.uniform(1, pr.PURPOSE_COARSE, P.nbcols * 3)
    assert vec_blockwise_rel_err(orc.spmv(A, x), A.to_scipy().tocsr() @ x, 2) < 1e-13
    assert vec_blockwise_rel_err(orc.spmv(P, xc), P.to_scipy().tocsr() @ xc, 2) < 1e-13
    assert vec_blockwise_rel_err(orc.spmv_t(P, x), P.to_scipy().tocsr().T @ x, 3) < 1e-13


def test_adjoint_identity(cfg0):
    # (P^T x) . y_c = x . (P y_c)
    P = cfg0.P(0)
    x = pr.uniform(0, pr.PURPOSE_FINE, P.nbrows * 3)
    yc = pr.uniform(0, pr.PURPOSE_COARSE, P.nbcols * 6)
    assert np.dot(orc.spmv_t(P, x), yc) == pytest.approx(np.dot(x, orc.spmv(P, yc)), rel=1e-13)


def test_transpose_explicit(cfg0):
    P = cfg0.P(0)
    R = orc.transpose(P)
    assert (R.nbrows, R.nbcols, R.bs_r, R.bs_c) == (P.nbcols, P.nbrows, 6, 3)
    Rd = pr.HostBSR(R.nbrows, R.nbcols, R.bs_r, R.bs_c, R.rowptr, R.colidx, R.vals).to_dense()
    assert (Rd == P.to_dense().T).all()
    for I in range(R.nbrows):
        assert (np.diff(R.colidx[R.rowptr[I]:R.rowptr[I + 1]]) > 0).all()
    assert np.diff(R.rowptr).max() == 125   # SURVEY master table: max blocks in a row of R, config 0


# ---------------------------------------------------------------- symbolic (I11)
def test_symbolic_counts_cfg0(cfg0):
    (rap, cap), (rc, cc) = orc.ptap_symbolic(cfg0.A(0), cfg0.P(0))
    assert cap.shape[0] == 4913 and cc.shape[0] == 343       # SURVEY master table (17^3, 7^3)
    assert np.diff(rap).max() == 27 and np.diff(rc).max() == 27
    for i in range(0, rap.shape[0] - 1, 37):
        assert (np.diff(cap[rap[i]:rap[i + 1]]) > 0).all()


def test_symbolic_vs_library_boolean_product(grid2d):
    import scipy.sparse as sp
    A, P = grid2d.A(0), grid2d.P(0)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    SA = sp.csr_matrix((np.ones(A.nnzb), A.colidx, A.rowptr), shape=(A.nbrows, A.nbcols))
    SP = sp.csr_matrix((np.ones(P.nnzb), P.colidx, P.rowptr), shape=(P.nbrows, P.nbcols))
    SAP = (SA @ SP).tocsr(); SAP.sort_indices()
    SAC = (SP.T @ SAP).tocsr(); SAC.sort_indices()
    assert (SAP.indptr == rap).all() and (SAP.indices == cap).all()
    assert (SAC.indptr == rc).all() and (SAC.indices == cc).all()


def test_symbolic_counts_closed_form_2d():
    # I11: tensor-product closed forms at config 1's shape, on a smaller grid with the same rule:
    # n = 3*na nodes per side: nnzb(A_c) = (3 na - 2)^2, nnzb(P) = (n + 2(na-1))^2... checked by the 1-D count
    ne = 47                                  # n = 48 = 3*16
    g = pr.Generator(2, ne, seed=1); g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    (rap, cap), (rc, cc) = orc.ptap_symbolic(A, P)
    n, na = ne + 1, (ne + 1) // 3
    p1d = sum(len({min(max(j, 0), n - 1) // 3 for j in (i - 1, i, i + 1)}) for i in range(n))
    assert P.nnzb == p1d ** 2
    ap1d = sum(len({min(max(j, 0), n - 1) // 3 for j in range(i - 2, i + 3)}) for i in range(n))
    assert cap.shape[0] == ap1d ** 2
    assert cc.shape[0] == (3 * na - 2) ** 2


# ---------------------------------------------------------------- PtAP numeric (I6, I7, I8, I9)
@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_ptap_vs_dense_brute_force(fix, request):
    # I8 (A_c = P^T A P): dense triple product by brute force equals forms 1 and 2
    g = request.getfixturevalue(fix)
    A, P = g.A(0), g.P(0)
    Ac1 = orc.ptap(A, P)
    dense = P.to_dense().T @ A.to_dense() @ P.to_dense()
    ref = dense_blocks(dense, Ac1.rowptr, Ac1.colidx, P.bs_c, P.bs_c)
    assert blockwise_rel_err(Ac1.vals, ref) < 1e-13
    # the symbolic pattern covers every non-zero of the dense product
    mask = np.zeros_like(dense, dtype=bool)
    for I in range(Ac1.nbrows):
        for k in range(Ac1.rowptr[I], Ac1.rowptr[I + 1]):
            J = Ac1.colidx[k]
            mask[I * P.bs_c:(I + 1) * P.bs_c, J * P.bs_c:(J + 1) * P.bs_c] = True
    assert np.abs(dense[~mask]).max(initial=0.0) == 0.0
    f2 = orc.PtapForm2(A, P)
    Ac2 = f2.run()
    assert blockwise_rel_err(Ac2.vals, ref) < 1e-13
    # AP materialised by form 2 equals the dense A P
    APd = A.to_dense() @ P.to_dense()
    Sd = np.abs(A.to_dense()) @ np.abs(P.to_dense())     # cancellation scale (structurally kept zero blocks)
    assert blockwise_rel_err(f2.vals_ap, dense_blocks(APd, f2.rap, f2.cap, A.bs_r, P.bs_c),
                             dense_blocks(Sd, f2.rap, f2.cap, A.bs_r, P.bs_c)) < 1e-13


def test_ptap_vs_scipy_library():
    g = pr.Generator(3, 12, seed=11); g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = orc.ptap(A, P)
    lib = (P.to_scipy().T @ A.to_scipy() @ P.to_scipy()).toarray()
    assert blockwise_rel_err(Ac.vals, dense_blocks(lib, Ac.rowptr, Ac.colidx, 6, 6)) < 1e-13


def test_ptap_selected_rows(cfg0):
    A, P = cfg0.A(0), cfg0.P(0)
    full = orc.ptap(A, P)
    part = orc.ptap(A, P, rows=[0, 13, 26])
    for I in (0, 13, 26):
        s = slice(full.rowptr[I], full.rowptr[I + 1])
        assert (part.vals[s] == full.vals[s]).all()
    assert (part.vals[full.rowptr[1]:full.rowptr[13]] == 0).all()


def test_coarse_operator_symmetric_spd(cfg0):
    # I7
    Ac = orc.ptap(cfg0.A(0), cfg0.P(0))
    D = pr.HostBSR(Ac.nbrows, Ac.nbcols, 6, 6, Ac.rowptr, Ac.colidx, Ac.vals).to_dense()
    assert np.abs(D - D.T).max() < 1e-15 * np.abs(D).max() * 10
    assert np.linalg.eigvalsh(D).min() > 0


def test_coarse_operator_keeps_near_null_space():
    # I6: Neumann problem, A_c B_coarse = 0
    g = pr.Generator(3, 8, seed=0, dirichlet=False)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    Ac = orc.ptap(A, P)
    c1 = g.level_arrays(1)
    Bc = np.zeros((P.nbcols * 6, 6))
    for J in range(P.nbcols):
        Mfull = np.eye(6)
        Mfull[:3, :] = rigid_modes(c1["coords"][J:J + 1], 3)
        Bc[J * 6:(J + 1) * 6] = c1["rfac"][J] @ Mfull
    Acd = pr.HostBSR(Ac.nbrows, Ac.nbcols, 6, 6, Ac.rowptr, Ac.colidx, Ac.vals).to_scipy()
    assert np.abs(Acd @ Bc).max() < 1e-14 * max(1.0, np.abs(Ac.vals).max()) * 10


def test_recompute_scaling_closed_form(cfg0):
    # I9 (config 2's protocol, reading R13): A_k = s_k A_0  =>  A_c^(k) = s_k A_c^(0)
    A, P = cfg0.A(0), cfg0.P(0)
    s = pr.uniform(2, pr.PURPOSE_RESCALE, 3, 0.5, 2.0)
    base = orc.ptap(A, P)
    f2 = orc.PtapForm2(A, P)
    for sk in s:
        Ak = pr.HostBSR(A.nbrows, A.nbcols, 3, 3, A.rowptr, A.colidx, A.vals * sk)
        assert blockwise_rel_err(orc.ptap(Ak, P, structure=(base.rowptr, base.colidx)).vals, sk * base.vals) < 1e-14
        assert blockwise_rel_err(f2.run(A.vals * sk).vals, sk * base.vals) < 1e-14


# ---------------------------------------------------------------- V-cycle and PCG (I12)
def _hier(g, nlev=2):
    A, P = g.A(0), g.P(0)
    Ac = orc.ptap(A, P)
    lam = g.level_info(0)["lam"]
    return A, P, Ac, lam


def cheb_poly_closed_form(A, Dinv, lam, lo=0.1, hi=1.1):
    """Error-propagation polynomial of the degree-2 Chebyshev smoother in closed form:
    p(t) = T_2((theta - t)/delta) / T_2(theta/delta), T_2(s) = 2 s^2 - 1.  Smoother: x <- x + (I - p(D^-1A)) A^-1 (b - A x)."""
    lmin, lmax = lo * lam, hi * lam
    theta, delta = (lmax + lmin) / 2, (lmax - lmin) / 2
    n = A.shape[0]
    T = (theta * np.eye(n) - Dinv @ A) / delta
    pA = (2 * T @ T - np.eye(n)) / (2 * (theta / delta) ** 2 - 1)
    return pA


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_chebyshev_smoother_closed_form(fix, request):
    g = request.getfixturevalue(fix)
    A, P, Ac, lam = _hier(g)
    H = orc.Hierarchy([A, Ac], [P], [lam])
    Ad = A.to_dense()
    bs = A.bs_r
    Dinv = np.zeros_like(Ad)
    for i in range(0, Ad.shape[0], bs):
        Dinv[i:i + bs, i:i + bs] = np.linalg.inv(Ad[i:i + bs, i:i + bs])
    pA = cheb_poly_closed_form(Ad, Dinv, lam)
    b = pr.uniform(g.seed, pr.PURPOSE_RHS, Ad.shape[0])
    x0 = pr.uniform(g.seed, pr.PURPOSE_FINE, Ad.shape[0])
    xs = np.linalg.solve(Ad, b)
    # error after smoothing = p(D^-1 A) * error before
    x1 = H.smooth(0, b, x0)
    ref = xs - pA @ (xs - x0)
    assert np.linalg.norm(x1 - ref) < 1e-12 * np.linalg.norm(ref)


@pytest.mark.parametrize("fix", ["cfg0", "grid2d"])
def test_two_grid_operator_dense(fix, request):
    # V-cycle assembled densely from its definition with the closed-form smoother
    g = request.getfixturevalue(fix)
    A, P, Ac, lam = _hier(g)
    H = orc.Hierarchy([A, Ac], [P], [lam])
    Ad, Pd = A.to_dense(), P.to_dense()
    bs = A.bs_r
    n = Ad.shape[0]
    Dinv = np.zeros_like(Ad)
    for i in range(0, n, bs):
        Dinv[i:i + bs, i:i + bs] = np.linalg.inv(Ad[i:i + bs, i:i + bs])
    S = (np.eye(n) - cheb_poly_closed_form(Ad, Dinv, lam)) @ np.linalg.inv(Ad)   # x <- x + S (b - A x)
    Acd = Pd.T @ Ad @ Pd
    b = pr.uniform(g.seed, pr.PURPOSE_RHS, n)
    x1 = S @ b
    x2 = x1 + Pd @ np.linalg.solve(Acd, Pd.T @ (b - Ad @ x1))
    x3 = x2 + S @ (b - Ad @ x2)
    got = H.vcycle(b)
    assert np.linalg.norm(got - x3) < 1e-11 * np.linalg.norm(x3)
    # I12: the V-cycle is a symmetric operator
    u = pr.uniform(g.seed, pr.PURPOSE_FINE, n)
    assert np.dot(u, H.vcycle(b)) == pytest.approx(np.dot(b, H.vcycle(u)), rel=1e-10)


def test_one_level_vcycle_is_direct_solve(grid2d):
    A = grid2d.A(0)
    H = orc.Hierarchy([A], [], [])
    b = pr.uniform(3, pr.PURPOSE_RHS, A.nbrows * 2)
    ref = np.linalg.solve(A.to_dense(), b)
    assert np.linalg.norm(H.vcycle(b) - ref) < 1e-11 * np.linalg.norm(ref)
    # PCG with the exact inverse as preconditioner converges in one iteration
    x, hist = H.pcg(b, 2)
    assert hist[0] == pytest.approx(np.linalg.norm(b), rel=1e-14)
    assert hist[1] < 1e-11 * hist[0]


def test_pcg_history_vs_dense_reference(cfg0):
    # PCG (unpreconditioned residual norm) against a dense numpy PCG using the V-cycle as an
    # explicit matrix M^-1; monotone decrease at roughly 0.3 per iteration (I12)
    A, P, Ac, lam = _hier(cfg0)
    H = orc.Hierarchy([A, Ac], [P], [lam])
    Ad = A.to_dense()
    n = Ad.shape[0]
    Minv = np.column_stack([H.vcycle(e) for e in np.eye(n)])
    b = pr.uniform(0, pr.PURPOSE_RHS, n)
    x, hist = H.pcg(b, 12)
    xr = np.zeros(n); r = b.copy(); z = Minv @ r; p = z.copy(); rz = r @ z
    ref = [np.linalg.norm(r)]
    for _ in range(12):
        q = Ad @ p
        a = rz / (p @ q)
        xr += a * p; r -= a * q
        ref.append(np.linalg.norm(r))
        z = Minv @ r
        rz_new = r @ z
        p = z + (rz_new / rz) * p
        rz = rz_new
    assert np.allclose(hist, ref, rtol=1e-7)
    assert (np.diff(hist) < 0).all()
    assert (hist[-1] / hist[0]) ** (1 / 12) < 0.5
    assert np.linalg.norm(Ad @ x - b) == pytest.approx(hist[-1], rel=1e-6)


# ---------------------------------------------------------------- three levels (O9, O10): the intermediate level
def _three_level(d, ne, seed):
    """A small three-level hierarchy built the way config 4 is (O9): A_1 = P_0^T A_0 P_0, level-2 prolongator from
    the restricted rigid-body modes, A_2 = P_1^T A_1 P_1."""
    g = pr.Generator(d, ne, seed=seed)
    g.build_prolongator(0)
    A0, P0 = g.A(0), g.P(0)
    Ac = orc.ptap(A0, P0)
    A1 = pr.HostBSR(Ac.nbrows, Ac.nbcols, Ac.bs_r, Ac.bs_c, Ac.rowptr, Ac.colidx, Ac.vals)
    g.set_operator(1, A1)
    g.build_prolongator(1)
    P1 = g.P(1)
    Ac2 = orc.ptap(A1, P1)
    A2 = pr.HostBSR(Ac2.nbrows, Ac2.nbcols, Ac2.bs_r, Ac2.bs_c, Ac2.rowptr, Ac2.colidx, Ac2.vals)
    lams = [g.level_info(0)["lam"], g.level_info(1)["lam"]]
    return g, [A0, A1, A2], [P0, P1], lams


def _dense_smoother(Ad, bs, lam):
    n = Ad.shape[0]
    Dinv = np.zeros_like(Ad)
    for i in range(0, n, bs):
        Dinv[i:i + bs, i:i + bs] = np.linalg.inv(Ad[i:i + bs, i:i + bs])     # library inverse of each bs x bs block
    return (np.eye(n) - cheb_poly_closed_form(Ad, Dinv, lam)) @ np.linalg.inv(Ad), Dinv


@pytest.mark.parametrize("d,ne", [(3, 8), (2, 26)])
def test_three_grid_operator_dense(d, ne):
    """PAPER.md:42 written out densely for THREE grids: the middle level both smooths (6x6 / 3x3 block-Jacobi,
    blocks inverted by numpy) and recurses.  Fails if vcycle() takes a level's operator, prolongator, lambda or
    D^-1 from the wrong level, or if the 6x6 block inverse is wrong."""
    g, As, Ps, lams = _three_level(d, ne, seed=21)
    assert As[1].bs_r == (6 if d == 3 else 3) and As[2].nbrows >= 1
    H = orc.Hierarchy(As, Ps, lams)
    A0, A1, A2 = (M.to_dense() for M in As)
    P0, P1 = (M.to_dense() for M in Ps)
    S0, _ = _dense_smoother(A0, As[0].bs_r, lams[0])
    S1, Dinv1 = _dense_smoother(A1, As[1].bs_r, lams[1])
    assert abs(lams[0] - lams[1]) > 1e-3 * lams[0]          # the two levels are distinguishable

    def level1(rc):                                          # V-cycle on level 1 from a zero guess
        y1 = S1 @ rc
        y2 = y1 + P1 @ np.linalg.solve(A2, P1.T @ (rc - A1 @ y1))
        return y2 + S1 @ (rc - A1 @ y2)

    b = pr.uniform(21, pr.PURPOSE_RHS, A0.shape[0])
    x1 = S0 @ b
    x2 = x1 + P0 @ level1(P0.T @ (b - A0 @ x1))
    x3 = x2 + S0 @ (b - A0 @ x2)
    got = H.vcycle(b)
    assert np.linalg.norm(got - x3) < 1e-10 * np.linalg.norm(x3)
    # the level-1 smoother on its own: error propagation p(D_1^-1 A_1) with numpy's 6x6 (3x3) inverses
    bc = pr.uniform(21, pr.PURPOSE_COARSE, A1.shape[0])
    y0 = pr.uniform(22, pr.PURPOSE_COARSE, A1.shape[0])
    ys = np.linalg.solve(A1, bc)
    ref = ys - cheb_poly_closed_form(A1, Dinv1, lams[1]) @ (ys - y0)
    y1 = H.smooth(1, bc, y0)
    assert np.linalg.norm(y1 - ref) < 1e-11 * np.linalg.norm(ref)
    # symmetric operator (I12), three levels
    u = pr.uniform(23, pr.PURPOSE_FINE, A0.shape[0])
    assert np.dot(u, got) == pytest.approx(np.dot(b, H.vcycle(u)), rel=1e-9)


def test_three_level_pcg_vs_dense_reference():
    g, As, Ps, lams = _three_level(2, 26, seed=5)
    H = orc.Hierarchy(As, Ps, lams)
    Ad = As[0].to_dense()
    n = Ad.shape[0]
    Minv = np.column_stack([H.vcycle(e) for e in np.eye(n)])
    assert np.abs(Minv - Minv.T).max() < 1e-9 * np.abs(Minv).max()
    b = pr.uniform(5, pr.PURPOSE_RHS, n)
    x, hist = H.pcg(b, 10)
    r = b.copy(); z = Minv @ r; p = z.copy(); rz = r @ z
    ref = [np.linalg.norm(r)]
    for _ in range(10):
        q = Ad @ p
        a = rz / (p @ q)
        r -= a * q
        ref.append(np.linalg.norm(r))
        z = Minv @ r
        rz_new = r @ z
        p = z + (rz_new / rz) * p
        rz = rz_new
    assert np.allclose(hist, ref, rtol=1e-7)
    assert (np.diff(hist) < 0).all()
