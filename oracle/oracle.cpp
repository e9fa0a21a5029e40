// oracle.cpp -- CPU reference ("oracle") for the blocked AMG hot path.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
// library.  It shares no code, header, table or helper with the CUDA path (paper_2606_24748_b200/csrc) and
// neither includes the other.  Plain, slow, obviously-correct C++17: every routine is the definition of the
// quantity written out, in the paper's notation, with no blocking, fusion or reordering.
//
// What the path computes (exactly, up to rounding order), and the passage that defines it:
//   orc_spmv            y = A x over stored bs_r x bs_c blocks
//   orc_spmv_t          y = A^T x  (restriction with R = P^T)               PAPER.md:42 ("restriction operator R")
//   orc_transpose       explicit R = P^T, rows sorted                       PAPER.md:103 ("the transpose R")
//   orc_spgemm_symbolic boolean product pattern, columns ascending          PAPER.md:80-82 ("reused sparsity")
//   orc_ptap_form1      A_c = P^T A P, row-by-row triple loop               PAPER.md:42, 58 (A_c = P^T A P)
//   orc_ptap_form2      the same through a materialised AP and R (timed)    PAPER.md:103 ("local blocked triple product")
//   orc_hier_*          block-Jacobi/Chebyshev V-cycle and PCG              PAPER.md:42 (cycle), 113 (pbjacobi, CG,
//                                                                           unpreconditioned residual norm)
//   orc_power_lambda    lambda of D^-1 A by 20 power iterations (omega = 4/(3 lambda))   PAPER.md:54-56; reading R10
//   orc_prolongator_smooth  P = (I - omega D^-1 A) P~ over the pattern of A P~   PAPER.md:54-56 (eq.), 244 (block AXPY
//                                                                           with SUBSET_NONZERO_PATTERN)
//   orc_bcoo_structure / orc_bcoo_sum   blocked COO assembly: coordinates declared once incl. duplicates, the value
//                       stream of dense bs_r x bs_c blocks summed per destination
// Floating point: fp64 data ("int32 indices and fp64 values"); sums that define one output
// entry are accumulated in long double and rounded once (reading R14), except form2 and the
// dense Cholesky, which use plain double (form2 is the timed CPU baseline).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): dense matvec / dense P^T A P by brute force at config 0
// and a 2D grid; scipy.sparse BSR products; adjoint identity; closed-form structure counts; A_c symmetry and
// rigid-body-mode annihilation; A_c^(k) = s_k A_c^(0); closed-form Chebyshev polynomial; two-grid operator
// assembled densely (two and three levels, 6x6 smoother blocks); V-cycle symmetry; PCG with exact preconditioner;
// prolongator smoothing against the dense formula, the generator's own P and exact mode reproduction on a Neumann
// problem; blocked COO against scipy's coordinate-format duplicate summation and a dense scatter-add.
// No routine here is "parity unpinned".
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
typedef struct {
  int32_t nbrows, nbcols, bs_r, bs_c;
  int64_t nnzb;
  const int32_t* rowptr;
  const int32_t* colidx;
  const double* vals;  // row-major inside a block, blocks in CSR order
} orc_bsr;
}

namespace {
typedef long double ld;

// y = A x by definition: y[i*bs_r + r] = sum_k sum_c A_k[r][c] * x[col(k)*bs_c + c]
void spmv(const orc_bsr& A, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int32_t i = 0; i < A.nbrows; ++i)
    for (int r = 0; r < A.bs_r; ++r) {
      ld s = 0;
      for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
        const double* blk = A.vals + (size_t)k * A.bs_r * A.bs_c;
        const double* xv = x + (size_t)A.colidx[k] * A.bs_c;
        for (int c = 0; c < A.bs_c; ++c) s += (ld)blk[r * A.bs_c + c] * (ld)xv[c];
      }
      y[(size_t)i * A.bs_r + r] = (double)s;
    }
}

// y = A^T x by definition: y[col(k)*bs_c + c] = sum over stored blocks of A_k[r][c] * x[i*bs_r + r]
void spmv_t(const orc_bsr& A, const double* x, double* y) {
  std::vector<ld> acc((size_t)A.nbcols * A.bs_c, 0.0L);
  for (int32_t i = 0; i < A.nbrows; ++i)
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const double* blk = A.vals + (size_t)k * A.bs_r * A.bs_c;
      for (int r = 0; r < A.bs_r; ++r)
        for (int c = 0; c < A.bs_c; ++c)
          acc[(size_t)A.colidx[k] * A.bs_c + c] += (ld)blk[r * A.bs_c + c] * (ld)x[(size_t)i * A.bs_r + r];
    }
  for (size_t t = 0; t < acc.size(); ++t) y[t] = (double)acc[t];
}

double dot(int64_t n, const double* a, const double* b) {
  ld s = 0;
  for (int64_t i = 0; i < n; ++i) s += (ld)a[i] * (ld)b[i];
  return (double)s;
}

// ------------------------------------------------------------------ hierarchy for the V-cycle (O10)
struct LevelData {
  orc_bsr A{}, P{};
  bool haveA = false, haveP = false;
  double lambda = 0;
  std::vector<double> Dinv;  // bs x bs per block row
};
struct Hier {
  int nlevels = 0, cheb_degree = 2;
  double lo = 0.1, hi = 1.1;
  std::vector<LevelData> L;
  std::vector<double> chol;  // dense lower Cholesky factor of the coarsest operator, n x n row-major
  int64_t ncoarse = 0;
};

bool invert_block(int n, const double* a, double* inv) {
  ld M[6][12];
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) { M[i][j] = a[i * n + j]; M[i][n + j] = (i == j); }
  for (int c = 0; c < n; ++c) {
    int p = c;
    for (int i = c + 1; i < n; ++i) if (fabsl(M[i][c]) > fabsl(M[p][c])) p = i;
    if (M[p][c] == 0) return false;
    if (p != c) for (int j = 0; j < 2 * n; ++j) std::swap(M[p][j], M[c][j]);
    const ld piv = M[c][c];
    for (int j = 0; j < 2 * n; ++j) M[c][j] /= piv;
    for (int i = 0; i < n; ++i) if (i != c) {
      const ld f = M[i][c];
      for (int j = 0; j < 2 * n; ++j) M[i][j] -= f * M[c][j];
    }
  }
  for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) inv[i * n + j] = (double)M[i][n + j];
  return true;
}

// z = D^-1 r, D the bs x bs block diagonal (point-block Jacobi)
void apply_dinv(const LevelData& lv, const double* r, double* z) {
  const int bs = lv.A.bs_r;
  for (int32_t i = 0; i < lv.A.nbrows; ++i)
    for (int a = 0; a < bs; ++a) {
      ld s = 0;
      for (int b = 0; b < bs; ++b) s += (ld)lv.Dinv[((size_t)i * bs + a) * bs + b] * (ld)r[(size_t)i * bs + b];
      z[(size_t)i * bs + a] = (double)s;
    }
}

// degree-k Chebyshev polynomial smoother in D^-1 A on [lo*lambda, hi*lambda] (reading R15):
//   theta=(lmax+lmin)/2, delta=(lmax-lmin)/2, sigma=theta/delta, rho_0=1/sigma
//   r=b-Ax; d_0=D^-1 r/theta; x+=d_0;
//   for k=1..deg-1: r-=A d_{k-1}; rho_k=1/(2 sigma-rho_{k-1}); d_k=rho_k rho_{k-1} d_{k-1}+(2 rho_k/delta) D^-1 r; x+=d_k
void chebyshev(const Hier& H, int l, const double* b, double* x) {
  const LevelData& lv = H.L[l];
  const int64_t n = (int64_t)lv.A.nbrows * lv.A.bs_r;
  const double lmin = H.lo * lv.lambda, lmax = H.hi * lv.lambda;
  const double theta = (lmax + lmin) / 2, delta = (lmax - lmin) / 2, sigma = theta / delta;
  std::vector<double> r(n), d(n), z(n), t(n);
  spmv(lv.A, x, t.data());
  for (int64_t i = 0; i < n; ++i) r[i] = b[i] - t[i];
  apply_dinv(lv, r.data(), z.data());
  for (int64_t i = 0; i < n; ++i) { d[i] = z[i] / theta; x[i] += d[i]; }
  double rho = 1 / sigma;
  for (int k = 1; k < H.cheb_degree; ++k) {
    spmv(lv.A, d.data(), t.data());
    for (int64_t i = 0; i < n; ++i) r[i] -= t[i];
    const double rho_new = 1 / (2 * sigma - rho);
    apply_dinv(lv, r.data(), z.data());
    for (int64_t i = 0; i < n; ++i) { d[i] = rho_new * rho * d[i] + (2 * rho_new / delta) * z[i]; x[i] += d[i]; }
    rho = rho_new;
  }
}

void chol_solve(const Hier& H, const double* b, double* x) {
  const int64_t n = H.ncoarse;
  const double* Lf = H.chol.data();
  std::vector<double> y(n);
  for (int64_t i = 0; i < n; ++i) {
    ld s = b[i];
    for (int64_t j = 0; j < i; ++j) s -= (ld)Lf[i * n + j] * (ld)y[j];
    y[i] = (double)(s / Lf[i * n + i]);
  }
  for (int64_t i = n - 1; i >= 0; --i) {
    ld s = y[i];
    for (int64_t j = i + 1; j < n; ++j) s -= (ld)Lf[j * n + i] * (ld)x[j];
    x[i] = (double)(s / Lf[i * n + i]);
  }
}

// one V-cycle from a zero initial guess: pre-smooth, residual, restrict, recurse, prolong + add,
// post-smooth; dense Cholesky solve on the coarsest level
void vcycle(const Hier& H, int l, const double* b, double* x) {
  const LevelData& lv = H.L[l];
  const int64_t n = (int64_t)lv.A.nbrows * lv.A.bs_r;
  if (l == H.nlevels - 1) { chol_solve(H, b, x); return; }
  for (int64_t i = 0; i < n; ++i) x[i] = 0;
  chebyshev(H, l, b, x);
  std::vector<double> r(n), t(n);
  spmv(lv.A, x, t.data());
  for (int64_t i = 0; i < n; ++i) r[i] = b[i] - t[i];
  const int64_t nc = (int64_t)lv.P.nbcols * lv.P.bs_c;
  std::vector<double> bc(nc), xc(nc);
  spmv_t(lv.P, r.data(), bc.data());
  vcycle(H, l + 1, bc.data(), xc.data());
  spmv(lv.P, xc.data(), t.data());
  for (int64_t i = 0; i < n; ++i) x[i] += t[i];
  chebyshev(H, l, b, x);
}

}  // namespace

// =================================================================== C ABI
extern "C" {

// threads the row-parallel routines use from now on (0: the OpenMP default); returns the count in effect.  Only the
// timing legs of bench.py call this (1 thread / all cores); it changes no arithmetic.
int orc_set_threads(int n) {
#ifdef _OPENMP
  static const int dflt = omp_get_max_threads();
  omp_set_num_threads(n > 0 ? n : dflt);
  return omp_get_max_threads();
#else
  (void)n;
  return 1;
#endif
}

int orc_spmv(const orc_bsr* A, const double* x, double* y) { spmv(*A, x, y); return 0; }
int orc_spmv_t(const orc_bsr* A, const double* x, double* y) { spmv_t(*A, x, y); return 0; }

// plain double, row-parallel: the timed CPU baseline of the SpMV family (same definition, double accumulator)
int orc_spmv_fast(const orc_bsr* Ap, const double* x, double* y) {
  const orc_bsr& A = *Ap;
#pragma omp parallel for schedule(static)
  for (int32_t i = 0; i < A.nbrows; ++i)
    for (int r = 0; r < A.bs_r; ++r) {
      double s = 0;
      for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
        const double* blk = A.vals + (size_t)k * A.bs_r * A.bs_c;
        const double* xv = x + (size_t)A.colidx[k] * A.bs_c;
        for (int c = 0; c < A.bs_c; ++c) s += blk[r * A.bs_c + c] * xv[c];
      }
      y[(size_t)i * A.bs_r + r] = s;
    }
  return 0;
}

// explicit transpose: T = A^T as BSR with bs_c x bs_r blocks, each block transposed, rows of T sorted by
// column (= ascending source row).  Caller allocates rowptr_t[nbcols+1], colidx_t[nnzb], vals_t[nnzb*bs_r*bs_c].
int orc_transpose(const orc_bsr* Ap, int32_t* rowptr_t, int32_t* colidx_t, double* vals_t) {
  const orc_bsr& A = *Ap;
  const int bb = A.bs_r * A.bs_c;
  for (int32_t j = 0; j <= A.nbcols; ++j) rowptr_t[j] = 0;
  for (int64_t k = 0; k < A.nnzb; ++k) rowptr_t[A.colidx[k] + 1]++;
  for (int32_t j = 0; j < A.nbcols; ++j) rowptr_t[j + 1] += rowptr_t[j];
  std::vector<int32_t> fill(rowptr_t, rowptr_t + A.nbcols);
  for (int32_t i = 0; i < A.nbrows; ++i)
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const int32_t q = fill[A.colidx[k]]++;
      colidx_t[q] = i;
      if (vals_t)
        for (int r = 0; r < A.bs_r; ++r)
          for (int c = 0; c < A.bs_c; ++c) vals_t[(size_t)q * bb + c * A.bs_r + r] = A.vals[(size_t)k * bb + r * A.bs_c + c];
    }
  return 0;
}

// boolean product pattern S_C = S_A * S_B (reading R5: symbolic, never dropped on value), columns
// strictly ascending.  Pass colidx_c = null to count only.  Returns nnzb(C); rowptr_c has nrows_a+1 entries.
int64_t orc_spgemm_symbolic(int32_t nrows_a, const int32_t* rowptr_a, const int32_t* colidx_a,
                            const int32_t* rowptr_b, const int32_t* colidx_b, int32_t* rowptr_c,
                            int32_t* colidx_c) {
  std::vector<int32_t> cols;
  int64_t n = 0;
  rowptr_c[0] = 0;
  for (int32_t i = 0; i < nrows_a; ++i) {
    cols.clear();
    for (int64_t k = rowptr_a[i]; k < rowptr_a[i + 1]; ++k) {
      const int32_t j = colidx_a[k];
      for (int64_t q = rowptr_b[j]; q < rowptr_b[j + 1]; ++q) cols.push_back(colidx_b[q]);
    }
    std::sort(cols.begin(), cols.end());
    cols.erase(std::unique(cols.begin(), cols.end()), cols.end());
    if (colidx_c) std::copy(cols.begin(), cols.end(), colidx_c + n);
    n += (int64_t)cols.size();
    rowptr_c[i + 1] = (int32_t)n;
  }
  return n;
}

// Form 1 (parity reference): A_c(I,J) = sum_i sum_j P(i,I)^T A(i,j) P(j,J), fine row by
// fine row: T_i(J) = sum_j A(i,j) P(j,J); then A_c(I,J) += P(i,I)^T T_i(J) for every stored P(i,I).
// Long double accumulators for A_c and T_i, rounded once at the end.  The structure (rowptr_c, colidx_c) is
// the symbolic one.  If nsel >= 0 only the coarse rows listed in sel[] are computed (the others are left
// untouched in vals_c) -- used for sampled full-size parity.
int orc_ptap_form1(const orc_bsr* Ap, const orc_bsr* Pp, const int32_t* rowptr_c, const int32_t* colidx_c,
                   double* vals_c, int32_t nsel, const int32_t* sel) {
  const orc_bsr &A = *Ap, &P = *Pp;
  if (A.bs_r != A.bs_c || A.bs_c != P.bs_r || A.nbcols != P.nbrows || A.nbrows != A.nbcols) return -1;
  const int bf = A.bs_r, bc = P.bs_c;
  const int32_t NC = P.nbcols;
  std::vector<char> want(NC, nsel < 0 ? 1 : 0);
  for (int32_t s = 0; s < (nsel < 0 ? 0 : nsel); ++s) want[sel[s]] = 1;
  // accumulators only for wanted rows
  std::vector<int64_t> accbase(NC + 1, 0);
  for (int32_t I = 0; I < NC; ++I) accbase[I + 1] = accbase[I] + (want[I] ? (int64_t)(rowptr_c[I + 1] - rowptr_c[I]) : 0);
  std::vector<ld> acc((size_t)accbase[NC] * bc * bc, 0.0L);
  std::vector<ld> T;            // dense row of AP over coarse block columns touched
  std::vector<int32_t> Tcols;   // the touched coarse columns, in first-touch order
  std::vector<int32_t> where(NC, -1);
  for (int32_t i = 0; i < A.nbrows; ++i) {
    bool need = false;
    for (int64_t q = P.rowptr[i]; q < P.rowptr[i + 1]; ++q) need = need || want[P.colidx[q]];
    if (!need) continue;
    Tcols.clear(); T.clear();
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const int32_t j = A.colidx[k];
      const double* a = A.vals + (size_t)k * bf * bf;
      for (int64_t q = P.rowptr[j]; q < P.rowptr[j + 1]; ++q) {
        const int32_t J = P.colidx[q];
        if (where[J] < 0) { where[J] = (int32_t)Tcols.size(); Tcols.push_back(J); T.resize(T.size() + (size_t)bf * bc, 0.0L); }
        ld* t = &T[(size_t)where[J] * bf * bc];
        const double* p = P.vals + (size_t)q * bf * bc;
        for (int r = 0; r < bf; ++r)
          for (int c = 0; c < bc; ++c)
            for (int m = 0; m < bf; ++m) t[r * bc + c] += (ld)a[r * bf + m] * (ld)p[m * bc + c];
      }
    }
    for (int64_t q = P.rowptr[i]; q < P.rowptr[i + 1]; ++q) {
      const int32_t I = P.colidx[q];
      if (!want[I]) continue;
      const double* pi = P.vals + (size_t)q * bf * bc;  // P(i,I), bf x bc
      for (size_t s = 0; s < Tcols.size(); ++s) {
        const int32_t J = Tcols[s];
        const int32_t* lo = colidx_c + rowptr_c[I];
        const int32_t* hi = colidx_c + rowptr_c[I + 1];
        const int32_t* it = std::lower_bound(lo, hi, J);
        if (it == hi || *it != J) return -2;  // structure does not contain the product pattern
        ld* out = &acc[(size_t)(accbase[I] + (it - lo)) * bc * bc];
        const ld* t = &T[s * bf * bc];
        for (int r = 0; r < bc; ++r)
          for (int c = 0; c < bc; ++c)
            for (int m = 0; m < bf; ++m) out[r * bc + c] += (ld)pi[m * bc + r] * t[m * bc + c];
      }
    }
    for (int32_t J : Tcols) where[J] = -1;
  }
  for (int32_t I = 0; I < NC; ++I) {
    if (!want[I]) continue;
    const int64_t nb = rowptr_c[I + 1] - rowptr_c[I];
    for (int64_t t = 0; t < nb * bc * bc; ++t)
      vals_c[(size_t)rowptr_c[I] * bc * bc + t] = (double)acc[(size_t)accbase[I] * bc * bc + t];
  }
  return 0;
}

// Form 2 (timed CPU baseline): materialise AP row-parallel over its symbolic structure, then
// A_c = R (AP) row-parallel with R = P^T given explicitly.  Plain double accumulators.
int orc_ptap_form2(const orc_bsr* Ap, const orc_bsr* Pp, const orc_bsr* Rp, const int32_t* rowptr_ap,
                   const int32_t* colidx_ap, double* vals_ap, const int32_t* rowptr_c, const int32_t* colidx_c,
                   double* vals_c) {
  const orc_bsr &A = *Ap, &P = *Pp, &R = *Rp;
  if (A.bs_r != A.bs_c || A.bs_c != P.bs_r || A.nbcols != P.nbrows) return -1;
  const int bf = A.bs_r, bc = P.bs_c;
  int bad = 0;
#pragma omp parallel for schedule(static)
  for (int32_t i = 0; i < A.nbrows; ++i) {
    const int32_t* lo = colidx_ap + rowptr_ap[i];
    const int32_t* hi = colidx_ap + rowptr_ap[i + 1];
    double* row = vals_ap + (size_t)rowptr_ap[i] * bf * bc;
    std::fill(row, row + (size_t)(hi - lo) * bf * bc, 0.0);
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const int32_t j = A.colidx[k];
      const double* a = A.vals + (size_t)k * bf * bf;
      for (int64_t q = P.rowptr[j]; q < P.rowptr[j + 1]; ++q) {
        const int32_t* it = std::lower_bound(lo, hi, P.colidx[q]);
        if (it == hi || *it != P.colidx[q]) { bad = 1; continue; }
        double* t = row + (size_t)(it - lo) * bf * bc;
        const double* p = P.vals + (size_t)q * bf * bc;
        for (int r = 0; r < bf; ++r)
          for (int c = 0; c < bc; ++c)
            for (int m = 0; m < bf; ++m) t[r * bc + c] += a[r * bf + m] * p[m * bc + c];
      }
    }
  }
#pragma omp parallel for schedule(static)
  for (int32_t I = 0; I < R.nbrows; ++I) {
    const int32_t* lo = colidx_c + rowptr_c[I];
    const int32_t* hi = colidx_c + rowptr_c[I + 1];
    double* row = vals_c + (size_t)rowptr_c[I] * bc * bc;
    std::fill(row, row + (size_t)(hi - lo) * bc * bc, 0.0);
    for (int64_t k = R.rowptr[I]; k < R.rowptr[I + 1]; ++k) {
      const int32_t i = R.colidx[k];
      const double* rb = R.vals + (size_t)k * bc * bf;  // R(I,i), bc x bf
      for (int64_t q = rowptr_ap[i]; q < rowptr_ap[i + 1]; ++q) {
        const int32_t* it = std::lower_bound(lo, hi, colidx_ap[q]);
        if (it == hi || *it != colidx_ap[q]) { bad = 1; continue; }
        double* out = row + (size_t)(it - lo) * bc * bc;
        const double* t = vals_ap + (size_t)q * bf * bc;
        for (int r = 0; r < bc; ++r)
          for (int c = 0; c < bc; ++c)
            for (int m = 0; m < bf; ++m) out[r * bc + c] += rb[r * bf + m] * t[m * bc + c];
      }
    }
  }
  return bad ? -2 : 0;
}

// ------------------------------------------------------------------ prolongator smoothing
// P = (I - omega D^-1 A) P~, D the bs x bs block diagonal of A (reading R11), on the
// boolean pattern of A*P~ (reading R5; the paper's MatAYPX adds P~ on a SUBSET of that pattern).
// Row by row, in the paper's order: T_i(J) = sum_j A(i,j) P~(j,J); P(i,J) = P~(i,J) - omega * D_i^-1 * T_i(J).
// Long double throughout (the inverse included), rounded once per entry.  (rowptr_p, colidx_p) is the symbolic
// pattern of A*P~ (orc_spgemm_symbolic); a P~ block outside it is an error.
int orc_prolongator_smooth(const orc_bsr* Ap, const orc_bsr* Ptp, double omega, const int32_t* rowptr_p,
                           const int32_t* colidx_p, double* vals_p) {
  const orc_bsr &A = *Ap, &Pt = *Ptp;
  if (A.bs_r != A.bs_c || A.nbrows != A.nbcols || A.nbcols != Pt.nbrows || A.bs_c != Pt.bs_r || A.bs_r > 6) return -1;
  const int bf = A.bs_r, bc = Pt.bs_c;
  int bad = 0;
#pragma omp parallel for schedule(static)
  for (int32_t i = 0; i < A.nbrows; ++i) {
    const int32_t* lo = colidx_p + rowptr_p[i];
    const int32_t* hi = colidx_p + rowptr_p[i + 1];
    const int64_t nslot = hi - lo;
    std::vector<ld> T((size_t)nslot * bf * bc, 0.0L);
    // D_i^-1 in long double (Gauss-Jordan with partial pivoting)
    ld M[6][12];
    bool found = false;
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k)
      if (A.colidx[k] == i) {
        for (int r = 0; r < bf; ++r)
          for (int c = 0; c < bf; ++c) { M[r][c] = A.vals[(size_t)k * bf * bf + r * bf + c]; M[r][bf + c] = (r == c); }
        found = true;
      }
    if (!found) { bad = 1; continue; }
    for (int c = 0; c < bf; ++c) {
      int p = c;
      for (int r = c + 1; r < bf; ++r) if (fabsl(M[r][c]) > fabsl(M[p][c])) p = r;
      if (M[p][c] == 0) { bad = 1; break; }
      if (p != c) for (int j = 0; j < 2 * bf; ++j) std::swap(M[p][j], M[c][j]);
      const ld piv = M[c][c];
      for (int j = 0; j < 2 * bf; ++j) M[c][j] /= piv;
      for (int r = 0; r < bf; ++r) if (r != c) {
        const ld f = M[r][c];
        for (int j = 0; j < 2 * bf; ++j) M[r][j] -= f * M[c][j];
      }
    }
    // T_i = row i of A * P~
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const int32_t j = A.colidx[k];
      const double* a = A.vals + (size_t)k * bf * bf;
      for (int64_t q = Pt.rowptr[j]; q < Pt.rowptr[j + 1]; ++q) {
        const int32_t* it = std::lower_bound(lo, hi, Pt.colidx[q]);
        if (it == hi || *it != Pt.colidx[q]) { bad = 1; continue; }
        ld* t = &T[(size_t)(it - lo) * bf * bc];
        const double* p = Pt.vals + (size_t)q * bf * bc;
        for (int r = 0; r < bf; ++r)
          for (int c = 0; c < bc; ++c)
            for (int m = 0; m < bf; ++m) t[r * bc + c] += (ld)a[r * bf + m] * (ld)p[m * bc + c];
      }
    }
    // P(i,J) = P~(i,J) - omega D_i^-1 T_i(J)
    for (int64_t s = 0; s < nslot; ++s) {
      const double* own = nullptr;
      for (int64_t q = Pt.rowptr[i]; q < Pt.rowptr[i + 1]; ++q)
        if (Pt.colidx[q] == lo[s]) own = Pt.vals + (size_t)q * bf * bc;
      for (int r = 0; r < bf; ++r)
        for (int c = 0; c < bc; ++c) {
          ld z = 0;
          for (int m = 0; m < bf; ++m) z += M[r][bf + m] * T[(size_t)s * bf * bc + m * bc + c];
          const ld v = (own ? (ld)own[r * bc + c] : 0.0L) - (ld)omega * z;
          vals_p[((size_t)rowptr_p[i] + s) * bf * bc + r * bc + c] = (double)v;
        }
    }
    // every P~ block of row i must lie inside the pattern (it does when A has its diagonal block)
    for (int64_t q = Pt.rowptr[i]; q < Pt.rowptr[i + 1]; ++q) {
      const int32_t* it = std::lower_bound(lo, hi, Pt.colidx[q]);
      if (it == hi || *it != Pt.colidx[q]) bad = 1;
    }
  }
  return bad ? -2 : 0;
}

// lambda of D^-1 A by power iteration (reading R10): v <- v0/||v0||_2; `iters` times: w = D^-1 (A v),
// lambda = ||w||_2, v = w / lambda; the last lambda is returned (omega = 4 / (3 lambda)).  D the
// bs x bs block diagonal (R11).  Long double sums.  Returns a negative value on a missing / singular diagonal block.
double orc_power_lambda(const orc_bsr* Ap, const double* v0, int iters) {
  const orc_bsr& A = *Ap;
  if (A.bs_r != A.bs_c || A.nbrows != A.nbcols || A.bs_r > 6) return -1.0;
  const int bs = A.bs_r;
  const int64_t n = (int64_t)A.nbrows * bs;
  std::vector<double> dinv((size_t)A.nbrows * bs * bs), v(v0, v0 + n), t(n), w(n);
  for (int32_t i = 0; i < A.nbrows; ++i) {
    bool ok = false;
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k)
      if (A.colidx[k] == i) { ok = invert_block(bs, A.vals + (size_t)k * bs * bs, &dinv[(size_t)i * bs * bs]); break; }
    if (!ok) return -2.0;
  }
  double nv = std::sqrt(dot(n, v.data(), v.data()));
  for (int64_t i = 0; i < n; ++i) v[i] /= nv;
  double lambda = 0.0;
  for (int it = 0; it < iters; ++it) {
    spmv(A, v.data(), t.data());
    for (int32_t i = 0; i < A.nbrows; ++i)
      for (int a = 0; a < bs; ++a) {
        ld sacc = 0;
        for (int b = 0; b < bs; ++b) sacc += (ld)dinv[((size_t)i * bs + a) * bs + b] * (ld)t[(size_t)i * bs + b];
        w[(size_t)i * bs + a] = (double)sacc;
      }
    lambda = std::sqrt(dot(n, w.data(), w.data()));
    for (int64_t i = 0; i < n; ++i) v[i] = w[i] / lambda;
  }
  return lambda;
}

// ------------------------------------------------------------------ blocked COO assembly
// the caller declares once the (block row, block column) coordinate of every contribution,
// duplicates included; the matrix has one block per distinct coordinate (rows in order, columns strictly ascending);
// every numeric assembly sums, per destination block, the dense bs_r x bs_c blocks of the value stream that carry
// its coordinate.  A contribution with a negative coordinate is ignored.  orc_bcoo_structure: pass colidx = null to
// count.  Returns nnzb, or -1 on a coordinate out of range.
int64_t orc_bcoo_structure(int64_t n, const int32_t* brow, const int32_t* bcol, int32_t nbrows, int32_t nbcols,
                           int32_t* rowptr, int32_t* colidx) {
  std::vector<std::vector<int32_t>> rows((size_t)nbrows);
  for (int64_t c = 0; c < n; ++c) {
    if (brow[c] < 0 || bcol[c] < 0) continue;   // declared but ignored (the COO convention for entries not owned)
    if (brow[c] >= nbrows || bcol[c] >= nbcols) return -1;
    rows[(size_t)brow[c]].push_back(bcol[c]);
  }
  int64_t nnzb = 0;
  rowptr[0] = 0;
  for (int32_t i = 0; i < nbrows; ++i) {
    std::vector<int32_t>& r = rows[(size_t)i];
    std::sort(r.begin(), r.end());
    r.erase(std::unique(r.begin(), r.end()), r.end());
    if (colidx) std::copy(r.begin(), r.end(), colidx + nnzb);
    nnzb += (int64_t)r.size();
    rowptr[i + 1] = (int32_t)nnzb;
  }
  return nnzb;
}

// vals[slot(brow[c], bcol[c])] += stream block c, for c = 0..n-1 in coordinate (declaration) order: a plain
// scatter-add, long double accumulators rounded once.  Returns -2 if a coordinate is not in the structure.
int orc_bcoo_sum(int64_t n, const int32_t* brow, const int32_t* bcol, const double* stream, int32_t bs_r,
                 int32_t bs_c, int32_t nbrows, const int32_t* rowptr, const int32_t* colidx, double* vals) {
  const int bb = bs_r * bs_c;
  const int64_t nnzb = rowptr[nbrows];
  std::vector<ld> acc((size_t)nnzb * bb, 0.0L);
  for (int64_t c = 0; c < n; ++c) {
    if (brow[c] < 0 || bcol[c] < 0) continue;
    const int32_t* lo = colidx + rowptr[brow[c]];
    const int32_t* hi = colidx + rowptr[brow[c] + 1];
    const int32_t* it = std::lower_bound(lo, hi, bcol[c]);
    if (it == hi || *it != bcol[c]) return -2;
    ld* a = &acc[(size_t)(it - colidx) * bb];
    for (int e = 0; e < bb; ++e) a[e] += (ld)stream[(size_t)c * bb + e];
  }
  for (size_t t = 0; t < acc.size(); ++t) vals[t] = (double)acc[t];
  return 0;
}

// ------------------------------------------------------------------ V-cycle / PCG (O10)
typedef struct Hier* orc_hier_t;

orc_hier_t orc_hier_create(int nlevels, int cheb_degree, double lo, double hi) {
  if (nlevels < 1) return nullptr;
  Hier* H = new Hier();
  H->nlevels = nlevels; H->cheb_degree = cheb_degree; H->lo = lo; H->hi = hi;
  H->L.resize(nlevels);
  return H;
}
void orc_hier_destroy(orc_hier_t H) { delete H; }

// arrays are borrowed: the caller keeps them alive.  P of level l maps level l+1 -> level l.
int orc_hier_set_level(orc_hier_t H, int l, const orc_bsr* A, const orc_bsr* P, double lambda) {
  if (!H || l < 0 || l >= H->nlevels || !A) return -1;
  H->L[l].A = *A; H->L[l].haveA = true;
  if (P) { H->L[l].P = *P; H->L[l].haveP = true; }
  H->L[l].lambda = lambda;
  return 0;
}

// D^-1 on every level (inverse of each bs x bs diagonal block) and the dense Cholesky factor of the coarsest
// operator (reading R17).  Call again after the operators' values change.
int orc_hier_setup(orc_hier_t H) {
  if (!H) return -1;
  for (int l = 0; l < H->nlevels; ++l) {
    LevelData& lv = H->L[l];
    if (!lv.haveA || (l < H->nlevels - 1 && !lv.haveP)) return -2;
    const int bs = lv.A.bs_r;
    lv.Dinv.assign((size_t)lv.A.nbrows * bs * bs, 0.0);
    for (int32_t i = 0; i < lv.A.nbrows; ++i) {
      bool ok = false;
      for (int64_t k = lv.A.rowptr[i]; k < lv.A.rowptr[i + 1]; ++k)
        if (lv.A.colidx[k] == i) { ok = invert_block(bs, lv.A.vals + (size_t)k * bs * bs, &lv.Dinv[(size_t)i * bs * bs]); break; }
      if (!ok) return -3;
    }
  }
  const orc_bsr& Ac = H->L[H->nlevels - 1].A;
  const int64_t n = (int64_t)Ac.nbrows * Ac.bs_r;
  const int bs = Ac.bs_r;
  H->ncoarse = n;
  H->chol.assign((size_t)n * n, 0.0);
  std::vector<double>& M = H->chol;
  for (int32_t i = 0; i < Ac.nbrows; ++i)
    for (int64_t k = Ac.rowptr[i]; k < Ac.rowptr[i + 1]; ++k)
      for (int r = 0; r < bs; ++r)
        for (int c = 0; c < bs; ++c)
          M[((size_t)i * bs + r) * n + (size_t)Ac.colidx[k] * bs + c] = Ac.vals[(size_t)k * bs * bs + r * bs + c];
  // Cholesky-Banachiewicz on the lower triangle, in place (textbook): L L^T = A
  for (int64_t j = 0; j < n; ++j) {
    double s = M[j * n + j];
    for (int64_t k = 0; k < j; ++k) s -= M[j * n + k] * M[j * n + k];
    if (!(s > 0)) return -4;
    const double ljj = std::sqrt(s);
    M[j * n + j] = ljj;
#pragma omp parallel for schedule(static)
    for (int64_t i = j + 1; i < n; ++i) {
      double t = M[i * n + j];
      for (int64_t k = 0; k < j; ++k) t -= M[i * n + k] * M[j * n + k];
      M[i * n + j] = t / ljj;
    }
  }
  for (int64_t i = 0; i < n; ++i)
    for (int64_t j = i + 1; j < n; ++j) M[i * n + j] = 0.0;
  return 0;
}

int orc_smooth(orc_hier_t H, int l, const double* b, double* x) {
  if (!H || l < 0 || l >= H->nlevels) return -1;
  chebyshev(*H, l, b, x);
  return 0;
}

// x = M^-1 b: one V-cycle from a zero initial guess
int orc_vcycle(orc_hier_t H, const double* b, double* x) {
  if (!H) return -1;
  vcycle(*H, 0, b, x);
  return 0;
}

// standard preconditioned CG, x_0 = 0, exactly `iters` iterations, hist[k] = ||r_k||_2 (unpreconditioned,
// PAPER.md:113), recursive residual update
int orc_pcg(orc_hier_t H, const double* b, double* x, int iters, double* hist) {
  if (!H) return -1;
  const orc_bsr& A = H->L[0].A;
  const int64_t n = (int64_t)A.nbrows * A.bs_r;
  std::vector<double> r(b, b + n), z(n), p(n), q(n);
  for (int64_t i = 0; i < n; ++i) x[i] = 0;
  hist[0] = std::sqrt(dot(n, r.data(), r.data()));
  vcycle(*H, 0, r.data(), z.data());
  p = z;
  double rz = dot(n, r.data(), z.data());
  for (int k = 0; k < iters; ++k) {
    spmv(A, p.data(), q.data());
    const double alpha = rz / dot(n, p.data(), q.data());
    for (int64_t i = 0; i < n; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
    hist[k + 1] = std::sqrt(dot(n, r.data(), r.data()));
    vcycle(*H, 0, r.data(), z.data());
    const double rz_new = dot(n, r.data(), z.data());
    const double beta = rz_new / rz;
    for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
    rz = rz_new;
  }
  return 0;
}

}  // extern "C"
