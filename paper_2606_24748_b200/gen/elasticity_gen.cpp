// elasticity_gen.cpp -- seeded synthetic-input generator (CPU, C++17, no dependencies).
//
// This module only MAKES INPUTS.  It is shared by the tests, the oracle-side checks and bench.py, and
// holds none of the hot path (SpMV family, PtAP symbolic/numeric, V-cycle, PCG): those live in
// paper_2606_24748_b200/csrc (CUDA) and, independently, in oracle/ (CPU).  Nothing here is included by
// either of them.
//
// What it builds (BASELINE.json configs; readings R3-R12, R20):
//   O1 mesh      unit square/cube, ne elements per side, n = ne+1 nodes, node id = ix + n*(iy + n*iz).
//   O2 element   Q1 isotropic linear elasticity (plane strain in 2D), 2-point Gauss per direction.
//   O3 assembly  block-CSR (BSR), bs = d, 3^d-point node stencil clipped to the grid, all structural
//                blocks kept ("dense bs x bs blocks that share a single index").
//   O4 Dirichlet face ix = 0: rows and columns zeroed, unit diagonal, structure kept (R4).
//   O5 boxes     3 nodes per direction, remainder merged into the last box (R6).
//   O6 P_tent    rigid-body modes about the aggregate centroid, Householder QR with diag(R) > 0
//                (near-null space represented exactly, bs 3 -> 6).
//   O7 smoothed  P = (I - omega D^-1 A) P_tent, D = block diagonal, omega = 4/(3 lambda), lambda from
//                20 power iterations on D^-1 A (R10, R11).
//   O9 level 2   coarse near-null space B_j(C) = R_j * M(c_j - C) (R9, R20).
// Random numbers: SplitMix64, one stream per (seed, purpose) (R12).
// Second workload: order = 2 builds the Q2 (triquadratic, 27-node hex /
// 9-node quad, 3-point Gauss) operator on the (2 ne + 1)^d node grid -- ~185 scalar nonzeros per row against Q1's ~78,
// the paper's Q2 harness has 169-180 -- and agg_mode = 1 replaces the node boxes by a seeded greedy disjoint covering
// of the operator's graph (root + neighbours, leftovers join an adjacent aggregate), which gives
// irregular aggregate sizes and coarse rows longer than the 27 of the box stencil.
//
// C ABI at the bottom (egen_*); all arrays are host memory owned by the handle.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

namespace {

// ---------------------------------------------------------------- random numbers (R12)
struct SplitMix64 {
  uint64_t s;
  uint64_t next() {
    uint64_t z = (s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  }
  double u01() { return (double)(next() >> 11) * 0x1.0p-53; }
};

// purposes: 0 power-iteration start (+16*level), 1 fine vector, 2 coarse vector, 3 right-hand side,
// 4 element moduli, 5 rescale factors.
SplitMix64 stream(uint64_t seed, uint64_t purpose) {
  SplitMix64 g{(seed + 1) * 0xD6E8FEB86659FD93ull ^ (purpose + 1) * 0xA0761D6478BD642Full};
  g.next();
  return g;
}

void fill_uniform(uint64_t seed, uint64_t purpose, int64_t n, double a, double b, double* out) {
  SplitMix64 g = stream(seed, purpose);
  for (int64_t i = 0; i < n; ++i) out[i] = a + (b - a) * g.u01();
}

// ---------------------------------------------------------------- containers
struct Bsr {
  int32_t nbrows = 0, nbcols = 0, bs_r = 0, bs_c = 0;
  std::vector<int32_t> rowptr, colidx;
  std::vector<double> vals;  // row-major inside a block, blocks in CSR order
  int64_t nnzb() const { return (int64_t)colidx.size(); }
};

struct Level {
  int d = 3;
  int nx[3] = {1, 1, 1};          // node grid of this level
  int bs = 3;                     // unknowns per node on this level
  int nb = 6;                     // near-null-space dimension = unknowns per node on the next level
  std::vector<double> coords;     // d per node (level >= 1: aggregate centroids)
  std::vector<double> Rfac;       // level >= 1: nb x nb R factor per node (row-major)
  Bsr A;
  bool haveA = false;
  // produced by build_P:
  Bsr Ptent, P;
  std::vector<int32_t> agg;       // node -> aggregate id
  double lambda = 0, omega = 0;
  bool haveP = false;
  int64_t nnodes() const { return (int64_t)nx[0] * nx[1] * nx[2]; }
};

struct Gen {
  int d = 3, ne = 8;
  double nu = 0.3;
  uint64_t seed = 0;
  int modulus_mode = 0;  // 0: E = 1; 1: per-element lognormal(0, 1) (config 3)
  int dirichlet = 1;     // 0: pure Neumann operator (used by the invariant tests)
  int order = 1;         // 1: Q1 elements, 2: Q2 elements (f4)
  int agg_mode = 0;      // 0: 3^d node boxes (R6), 1: seeded greedy disjoint covering of the graph (f4)
  std::vector<Level> levels;
  std::vector<double> Emod;  // per-element modulus (empty: 1 everywhere)
  std::vector<double> Ke;    // reference element matrix (E = 1)
  std::string err;
};

// ---------------------------------------------------------------- O2: element matrix
// K[(a*d+i)][(b*d+j)] = int  lam d_i N_a d_j N_b + mu d_j N_a d_i N_b + mu delta_ij grad N_a . grad N_b
// Tensor-product Lagrange element of order p (1: Q1, 2: Q2) on a cube of side h: local node a has index a_k in
// {0..p} in direction k, a = a_0 + (p+1) (a_1 + (p+1) a_2) (x fastest); p+1 Gauss points per direction.
void element_matrix(int d, int p, double h, double E, double nu, std::vector<double>& K) {
  const int n1 = p + 1;
  int nen = 1;
  for (int k = 0; k < d; ++k) nen *= n1;
  const int nd = d * nen;
  K.assign((size_t)nd * nd, 0.0);
  const double lam = E * nu / ((1 + nu) * (1 - 2 * nu)), mu = E / (2 * (1 + nu));
  double gp[3], gw[3];
  if (p == 1) { gp[0] = -1.0 / std::sqrt(3.0); gp[1] = -gp[0]; gw[0] = gw[1] = 1.0; }
  else { gp[0] = -std::sqrt(0.6); gp[1] = 0.0; gp[2] = std::sqrt(0.6); gw[0] = gw[2] = 5.0 / 9.0; gw[1] = 8.0 / 9.0; }
  auto shape = [&](int a, double xi, double& N, double& dN) {   // 1D Lagrange on nodes -1, (0,) 1
    if (p == 1) { const double s = a ? 1.0 : -1.0; N = (1 + s * xi) / 2; dN = s / 2; }
    else if (a == 0) { N = xi * (xi - 1) / 2; dN = xi - 0.5; }
    else if (a == 1) { N = 1 - xi * xi; dN = -2 * xi; }
    else { N = xi * (xi + 1) / 2; dN = xi + 0.5; }
  };
  const double detJ = std::pow(h / 2, d);
  int nq = 1;
  for (int k = 0; k < d; ++k) nq *= n1;
  std::vector<double> dN((size_t)nen * 3);
  for (int q = 0; q < nq; ++q) {
    double xi[3] = {0, 0, 0}, w = 1;
    for (int k = 0, t = q; k < d; ++k, t /= n1) { xi[k] = gp[t % n1]; w *= gw[t % n1]; }
    for (int a = 0; a < nen; ++a) {
      int ak[3] = {0, 0, 0};
      for (int k = 0, t = a; k < d; ++k, t /= n1) ak[k] = t % n1;
      for (int k = 0; k < d; ++k) {
        double v = 1;
        for (int m = 0; m < d; ++m) {
          double N, D;
          shape(ak[m], xi[m], N, D);
          v *= (m == k) ? D : N;
        }
        dN[(size_t)a * 3 + k] = v * (2 / h);
      }
    }
    for (int a = 0; a < nen; ++a)
      for (int b = 0; b < nen; ++b) {
        double gg = 0;
        for (int k = 0; k < d; ++k) gg += dN[(size_t)a * 3 + k] * dN[(size_t)b * 3 + k];
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) {
            double v = lam * dN[(size_t)a * 3 + i] * dN[(size_t)b * 3 + j] + mu * dN[(size_t)a * 3 + j] * dN[(size_t)b * 3 + i] +
                       (i == j ? mu * gg : 0.0);
            K[(size_t)(a * d + i) * nd + (b * d + j)] += v * detJ * w;
          }
      }
  }
}

// ---------------------------------------------------------------- O1, O3, O4: fine operator
// Node i (one direction) of an order-p grid couples to the nodes of the elements that contain it: an element-corner
// node (i % p == 0) to [i-p, i+p], an interior node to its own element [i - i%p, i - i%p + p]; clipped to the grid.
inline int nb_lo(int i, int p) { return std::max(0, i - ((i % p == 0) ? p : i % p)); }
inline int nb_hi(int i, int p, int n) { return std::min(n - 1, i + ((i % p == 0) ? p : p - i % p)); }
// elements containing node i: [el_lo, el_hi]
inline int el_lo(int i, int p) { return std::max(0, (i % p == 0) ? i / p - 1 : i / p); }
inline int el_hi(int i, int p, int ne) { return std::min(ne - 1, i / p); }

void build_fine_operator(Gen& G) {
  Level& L = G.levels[0];
  const int d = G.d, p = G.order, ne = G.ne, n = p * ne + 1, n1 = p + 1;
  L.d = d; L.bs = d; L.nb = (d == 3) ? 6 : 3;
  L.nx[0] = n; L.nx[1] = n; L.nx[2] = (d == 3) ? n : 1;
  const int nz = L.nx[2];
  const int64_t N = L.nnodes();
  const double h = 1.0 / ne, hn = h / p;
  L.coords.resize((size_t)N * d);
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        int64_t id = ix + (int64_t)n * (iy + (int64_t)n * iz);
        L.coords[id * d + 0] = ix * hn;
        L.coords[id * d + 1] = iy * hn;
        if (d == 3) L.coords[id * d + 2] = iz * hn;
      }
  // per-element Young's modulus (config 3: lognormal(0,1), Box-Muller cosine branch, element order)
  const int nez = (d == 3) ? ne : 1;
  const int64_t NE = (int64_t)ne * ne * nez;
  std::vector<double>& Emod = G.Emod;
  if (G.modulus_mode == 1) {
    Emod.resize(NE);
    SplitMix64 g = stream(G.seed, 4);
    for (int64_t e = 0; e < NE; ++e) {
      double u1 = 1.0 - g.u01(), u2 = g.u01();
      double z = std::sqrt(-2 * std::log(u1)) * std::cos(2 * M_PI * u2);
      Emod[e] = std::exp(z);
    }
  }
  std::vector<double>& Ke = G.Ke;
  element_matrix(d, p, h, 1.0, G.nu, Ke);
  int nen = 1;
  for (int k = 0; k < d; ++k) nen *= n1;
  const int nd = d * nen, bb = d * d;

  Bsr& A = L.A;
  A.nbrows = A.nbcols = (int32_t)N; A.bs_r = A.bs_c = d;
  A.rowptr.assign(N + 1, 0);
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        int64_t id = ix + (int64_t)n * (iy + (int64_t)n * iz);
        int cx = nb_hi(ix, p, n) - nb_lo(ix, p) + 1, cy = nb_hi(iy, p, n) - nb_lo(iy, p) + 1;
        int cz = (d == 3) ? nb_hi(iz, p, nz) - nb_lo(iz, p) + 1 : 1;
        A.rowptr[id + 1] = cx * cy * cz;
      }
  for (int64_t i = 0; i < N; ++i) A.rowptr[i + 1] += A.rowptr[i];
  const int64_t nnzb = A.rowptr[N];
  A.colidx.resize(nnzb);
  A.vals.assign((size_t)nnzb * bb, 0.0);

#pragma omp parallel for schedule(static) collapse(2)
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        const int64_t id = ix + (int64_t)n * (iy + (int64_t)n * iz);
        const int x0 = nb_lo(ix, p), y0 = nb_lo(iy, p), z0 = (d == 3) ? nb_lo(iz, p) : 0;
        const int cx = nb_hi(ix, p, n) - x0 + 1, cy = nb_hi(iy, p, n) - y0 + 1;
        const int cz = (d == 3) ? nb_hi(iz, p, nz) - z0 + 1 : 1;
        const int64_t base = A.rowptr[id];
        for (int sz = 0; sz < cz; ++sz)
          for (int sy = 0; sy < cy; ++sy)
            for (int sx = 0; sx < cx; ++sx)
              A.colidx[base + (sz * cy + sy) * cx + sx] =
                  (int32_t)((x0 + sx) + (int64_t)n * ((y0 + sy) + (int64_t)n * (z0 + sz)));
        // gather form of the element loop: adjacent elements in ascending element id
        const int ez0 = (d == 3) ? el_lo(iz, p) : 0, ez1 = (d == 3) ? el_hi(iz, p, ne) : 0;
        for (int ez = ez0; ez <= ez1; ++ez)
          for (int ey = el_lo(iy, p); ey <= el_hi(iy, p, ne); ++ey)
            for (int ex = el_lo(ix, p); ex <= el_hi(ix, p, ne); ++ex) {
              const int64_t e = ex + (int64_t)ne * (ey + (int64_t)ne * (d == 3 ? ez : 0));
              const double Ee = Emod.empty() ? 1.0 : Emod[e];
              const int a = (ix - p * ex) + n1 * ((iy - p * ey) + n1 * (d == 3 ? iz - p * ez : 0));
              for (int b = 0; b < nen; ++b) {
                const int bx = p * ex + b % n1, by = p * ey + (b / n1) % n1, bz = (d == 3) ? p * ez + b / (n1 * n1) : 0;
                const int64_t slot = base + ((bz - z0) * cy + (by - y0)) * cx + (bx - x0);
                double* blk = &A.vals[(size_t)slot * bb];
                for (int i = 0; i < d; ++i)
                  for (int j = 0; j < d; ++j) blk[i * d + j] += Ee * Ke[(size_t)(a * d + i) * nd + (b * d + j)];
              }
            }
        if (G.dirichlet) {  // O4
          for (int64_t k = base; k < A.rowptr[id + 1]; ++k) {
            const int64_t j = A.colidx[k];
            const bool ci = (ix == 0), cj = (j % n == 0);
            if (ci || cj) {
              double* blk = &A.vals[(size_t)k * bb];
              for (int t = 0; t < bb; ++t) blk[t] = 0.0;
              if (j == id)
                for (int i = 0; i < d; ++i) blk[i * d + i] = 1.0;
            }
          }
        }
      }
  L.haveA = true;
}

// ---------------------------------------------------------------- small dense helpers
// Thin Householder QR of B (m x n, row-major, m >= n): on exit Q (m x n) has orthonormal columns, R (n x n)
// is upper triangular with positive diagonal, Q R = B.
bool householder_qr(int m, int n, std::vector<double>& B, std::vector<double>& Q, std::vector<double>& R) {
  std::vector<double> V((size_t)m * n, 0.0), beta(n, 0.0);
  for (int k = 0; k < n; ++k) {
    double nrm = 0;
    for (int i = k; i < m; ++i) nrm += B[(size_t)i * n + k] * B[(size_t)i * n + k];
    nrm = std::sqrt(nrm);
    if (nrm == 0) return false;
    const double alpha = (B[(size_t)k * n + k] > 0) ? -nrm : nrm;
    double vnorm2 = 0;
    for (int i = k; i < m; ++i) {
      double v = B[(size_t)i * n + k] - (i == k ? alpha : 0.0);
      V[(size_t)i * n + k] = v;
      vnorm2 += v * v;
    }
    beta[k] = (vnorm2 > 0) ? 2.0 / vnorm2 : 0.0;
    for (int j = k; j < n; ++j) {
      double s = 0;
      for (int i = k; i < m; ++i) s += V[(size_t)i * n + k] * B[(size_t)i * n + j];
      s *= beta[k];
      for (int i = k; i < m; ++i) B[(size_t)i * n + j] -= s * V[(size_t)i * n + k];
    }
  }
  R.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int j = i; j < n; ++j) R[(size_t)i * n + j] = B[(size_t)i * n + j];
  Q.assign((size_t)m * n, 0.0);
  for (int j = 0; j < n; ++j) Q[(size_t)j * n + j] = 1.0;
  for (int k = n - 1; k >= 0; --k)
    for (int j = 0; j < n; ++j) {
      double s = 0;
      for (int i = k; i < m; ++i) s += V[(size_t)i * n + k] * Q[(size_t)i * n + j];
      s *= beta[k];
      for (int i = k; i < m; ++i) Q[(size_t)i * n + j] -= s * V[(size_t)i * n + k];
    }
  for (int k = 0; k < n; ++k)
    if (R[(size_t)k * n + k] < 0) {
      for (int j = 0; j < n; ++j) R[(size_t)k * n + j] = -R[(size_t)k * n + j];
      for (int i = 0; i < m; ++i) Q[(size_t)i * n + k] = -Q[(size_t)i * n + k];
    }
  return true;
}

// inverse of a small dense matrix (n <= 6) by Gauss-Jordan with partial pivoting; row-major
bool small_inverse(int n, const double* a, double* inv) {
  double M[6][12];
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) { M[i][j] = a[i * n + j]; M[i][n + j] = (i == j); }
  for (int c = 0; c < n; ++c) {
    int p = c;
    for (int i = c + 1; i < n; ++i) if (std::fabs(M[i][c]) > std::fabs(M[p][c])) p = i;
    if (M[p][c] == 0) return false;
    if (p != c) for (int j = 0; j < 2 * n; ++j) std::swap(M[p][j], M[c][j]);
    const double piv = 1.0 / M[c][c];
    for (int j = 0; j < 2 * n; ++j) M[c][j] *= piv;
    for (int i = 0; i < n; ++i) if (i != c) {
      const double f = M[i][c];
      if (f != 0) for (int j = 0; j < 2 * n; ++j) M[i][j] -= f * M[c][j];
    }
  }
  for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) inv[i * n + j] = M[i][n + j];
  return true;
}

// near-null-space block of one node about centre C: bs x nb, row-major
// level 0: [I | W(x - C)], W(r)[:,k] = e_k x r (3D); (-(y), x)^T in 2D.   level >= 1: R_j * M(c_j - C).
void nullspace_block(const Level& L, int64_t node, const double* C, double* out) {
  const int d = L.d, bs = L.bs, nb = L.nb;
  double r[3] = {0, 0, 0};
  for (int k = 0; k < d; ++k) r[k] = L.coords[node * d + k] - C[k];
  double M[36];
  for (int i = 0; i < nb * nb; ++i) M[i] = 0;
  for (int i = 0; i < nb; ++i) M[i * nb + i] = 1;
  if (d == 3) {
    const double W[3][3] = {{0, r[2], -r[1]}, {-r[2], 0, r[0]}, {r[1], -r[0], 0}};
    for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) M[i * nb + 3 + k] = W[i][k];
  } else {
    M[0 * nb + 2] = -r[1];
    M[1 * nb + 2] = r[0];
  }
  if (L.Rfac.empty()) {  // level 0: bs = d rows of [I | W]
    for (int i = 0; i < bs; ++i) for (int j = 0; j < nb; ++j) out[i * nb + j] = M[i * nb + j];
  } else {               // level >= 1: bs = nb
    const double* Rj = &L.Rfac[(size_t)node * nb * nb];
    for (int i = 0; i < nb; ++i)
      for (int j = 0; j < nb; ++j) {
        double s = 0;
        for (int k = 0; k < nb; ++k) s += Rj[i * nb + k] * M[k * nb + j];
        out[i * nb + j] = s;
      }
  }
}

// ---------------------------------------------------------------- O5-O7, O9: prolongator of one level
bool build_P(Gen& G, int l) {
  if ((int)G.levels.size() <= l + 1) G.levels.resize(l + 2);
  Level& L = G.levels[l];
  if (!L.haveA) { G.err = "level operator not set"; return false; }
  const int d = L.d, bs = L.bs, nb = L.nb;
  const int64_t N = L.nnodes();
  int na[3] = {1, 1, 1};
  int64_t NA = 0;
  L.agg.assign(N, -1);
  if (G.agg_mode == 0) {
    for (int k = 0; k < d; ++k) na[k] = std::max(1, L.nx[k] / 3);
    NA = (int64_t)na[0] * na[1] * na[2];
    for (int iz = 0; iz < L.nx[2]; ++iz)
      for (int iy = 0; iy < L.nx[1]; ++iy)
        for (int ix = 0; ix < L.nx[0]; ++ix) {
          const int64_t id = ix + (int64_t)L.nx[0] * (iy + (int64_t)L.nx[1] * iz);
          const int ax = std::min(ix / 3, na[0] - 1), ay = std::min(iy / 3, na[1] - 1);
          const int az = (d == 3) ? std::min(iz / 3, na[2] - 1) : 0;
          L.agg[id] = (int32_t)(ax + (int64_t)na[0] * (ay + (int64_t)na[1] * az));
        }
  } else {
    // greedy disjoint covering of the operator's graph, every stored block an edge (threshold 0):
    // pass 1 visits the nodes in a seeded random order and makes root + neighbours an aggregate when all of them
    // are still free; later passes attach every free node to the aggregate of its first aggregated neighbour, one
    // ring per pass (deterministic: decisions of a pass use the state before the pass)
    const Bsr& G0 = L.A;
    std::vector<int32_t> order(N);
    for (int64_t i = 0; i < N; ++i) order[i] = (int32_t)i;
    SplitMix64 g = stream(G.seed, 6 + 16 * (uint64_t)l);
    for (int64_t i = N - 1; i > 0; --i) std::swap(order[i], order[(int64_t)(g.next() % (uint64_t)(i + 1))]);
    for (int64_t t = 0; t < N; ++t) {
      const int32_t r = order[t];
      bool free_all = true;
      for (int64_t k = G0.rowptr[r]; k < G0.rowptr[r + 1] && free_all; ++k) free_all = L.agg[G0.colidx[k]] < 0;
      if (!free_all || L.agg[r] >= 0) continue;
      for (int64_t k = G0.rowptr[r]; k < G0.rowptr[r + 1]; ++k) L.agg[G0.colidx[k]] = (int32_t)NA;
      L.agg[r] = (int32_t)NA;
      ++NA;
    }
    if (NA == 0) { G.err = "empty graph"; return false; }
    for (bool left = true; left;) {
      left = false;
      std::vector<int32_t> next(L.agg);
      bool progress = false;
      for (int64_t i = 0; i < N; ++i) {
        if (L.agg[i] >= 0) continue;
        for (int64_t k = G0.rowptr[i]; k < G0.rowptr[i + 1]; ++k)
          if (L.agg[G0.colidx[k]] >= 0) { next[i] = L.agg[G0.colidx[k]]; progress = true; break; }
        if (next[i] < 0) left = true;
      }
      L.agg.swap(next);
      if (left && !progress) { G.err = "disconnected graph in aggregation"; return false; }
    }
    na[0] = (int)NA;
  }
  std::vector<std::vector<int32_t>> members(NA);
  for (int64_t id = 0; id < N; ++id) members[L.agg[id]].push_back((int32_t)id);  // ascending node id
  // next level skeleton
  Level& Lc = G.levels[l + 1];
  Level& Lf = L;
  Lc.d = d; Lc.bs = nb; Lc.nb = nb;
  Lc.nx[0] = na[0]; Lc.nx[1] = na[1]; Lc.nx[2] = na[2];
  Lc.coords.assign((size_t)NA * d, 0.0);
  Lc.Rfac.assign((size_t)NA * nb * nb, 0.0);
  Lc.haveA = false; Lc.haveP = false;

  // O6 / O9: tentative prolongator, one bs x nb block per fine node
  Bsr& Pt = Lf.Ptent;
  Pt.nbrows = (int32_t)N; Pt.nbcols = (int32_t)NA; Pt.bs_r = bs; Pt.bs_c = nb;
  Pt.rowptr.resize(N + 1);
  Pt.colidx.resize(N);
  Pt.vals.assign((size_t)N * bs * nb, 0.0);
  for (int64_t i = 0; i <= N; ++i) Pt.rowptr[i] = (int32_t)i;
  for (int64_t i = 0; i < N; ++i) Pt.colidx[i] = Lf.agg[i];
  bool ok = true;
#pragma omp parallel for schedule(static)
  for (int64_t J = 0; J < NA; ++J) {
    const auto& mem = members[J];
    const int m = (int)mem.size() * bs;
    double C[3] = {0, 0, 0};
    for (int32_t node : mem) for (int k = 0; k < d; ++k) C[k] += Lf.coords[(size_t)node * d + k];
    for (int k = 0; k < d; ++k) C[k] /= (double)mem.size();
    for (int k = 0; k < d; ++k) Lc.coords[J * d + k] = C[k];
    std::vector<double> B((size_t)m * nb), Q, R;
    for (size_t t = 0; t < mem.size(); ++t) nullspace_block(Lf, mem[t], C, &B[t * bs * nb]);
    if (m < nb || !householder_qr(m, nb, B, Q, R)) {
#pragma omp critical
      ok = false;
      continue;
    }
    for (size_t t = 0; t < mem.size(); ++t)
      std::memcpy(&Pt.vals[(size_t)mem[t] * bs * nb], &Q[t * bs * nb], sizeof(double) * bs * nb);
    std::memcpy(&Lc.Rfac[(size_t)J * nb * nb], R.data(), sizeof(double) * nb * nb);
  }
  if (!ok) { G.err = "rank-deficient aggregate in QR"; return false; }

  // O7: D^-1, lambda by 20 power iterations on D^-1 A (R10), omega = 4 / (3 lambda)
  const Bsr& A = Lf.A;
  const int bb = bs * bs;
  std::vector<double> Dinv((size_t)N * bb);
  ok = true;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    bool found = false;
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k)
      if (A.colidx[k] == i) { found = small_inverse(bs, &A.vals[(size_t)k * bb], &Dinv[(size_t)i * bb]); break; }
    if (!found) {
#pragma omp critical
      ok = false;
    }
  }
  if (!ok) { G.err = "singular or missing diagonal block"; return false; }
  const int64_t nu = N * bs;
  std::vector<double> v(nu), w(nu), t(nu);
  fill_uniform(G.seed, 0 + 16 * (uint64_t)l, nu, -1.0, 1.0, v.data());
  auto norm2 = [&](const std::vector<double>& x) {
    double s = 0;
    for (int64_t i = 0; i < nu; ++i) s += x[i] * x[i];
    return std::sqrt(s);
  };
  {
    const double nv = norm2(v);
    for (int64_t i = 0; i < nu; ++i) v[i] /= nv;
  }
  double lambda = 0;
  for (int it = 0; it < 20; ++it) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
      double acc[6] = {0, 0, 0, 0, 0, 0};
      for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
        const double* blk = &A.vals[(size_t)k * bb];
        const double* xv = &v[(size_t)A.colidx[k] * bs];
        for (int r = 0; r < bs; ++r) for (int c = 0; c < bs; ++c) acc[r] += blk[r * bs + c] * xv[c];
      }
      const double* Di = &Dinv[(size_t)i * bb];
      for (int r = 0; r < bs; ++r) {
        double s = 0;
        for (int c = 0; c < bs; ++c) s += Di[r * bs + c] * acc[c];
        w[i * bs + r] = s;
      }
    }
    lambda = norm2(w);
    for (int64_t i = 0; i < nu; ++i) v[i] = w[i] / lambda;
  }
  Lf.lambda = lambda;
  Lf.omega = 4.0 / (3.0 * lambda);

  // pattern of A * P_tent: row i -> sorted unique aggregates of the columns of row i
  Bsr& P = Lf.P;
  P.nbrows = (int32_t)N; P.nbcols = (int32_t)NA; P.bs_r = bs; P.bs_c = nb;
  P.rowptr.assign(N + 1, 0);
  std::vector<std::vector<int32_t>> rowcols(N);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    std::vector<int32_t>& c = rowcols[i];
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) c.push_back(Lf.agg[A.colidx[k]]);
    std::sort(c.begin(), c.end());
    c.erase(std::unique(c.begin(), c.end()), c.end());
  }
  for (int64_t i = 0; i < N; ++i) P.rowptr[i + 1] = P.rowptr[i] + (int32_t)rowcols[i].size();
  const int64_t pn = P.rowptr[N];
  P.colidx.resize(pn);
  P.vals.assign((size_t)pn * bs * nb, 0.0);
  const int pb = bs * nb;
  const double omega = Lf.omega;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    const int64_t p0 = P.rowptr[i];
    const int cnt = (int)rowcols[i].size();
    for (int s = 0; s < cnt; ++s) P.colidx[p0 + s] = rowcols[i][s];
    std::vector<double> T((size_t)cnt * pb, 0.0);  // row i of A * P_tent
    for (int64_t k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      const int64_t j = A.colidx[k];
      const int s = (int)(std::lower_bound(rowcols[i].begin(), rowcols[i].end(), Lf.agg[j]) - rowcols[i].begin());
      const double* a = &A.vals[(size_t)k * bb];
      const double* q = &Pt.vals[(size_t)j * pb];
      double* tt = &T[(size_t)s * pb];
      for (int r = 0; r < bs; ++r)
        for (int c = 0; c < nb; ++c) {
          double sum = 0;
          for (int m = 0; m < bs; ++m) sum += a[r * bs + m] * q[m * nb + c];
          tt[r * nb + c] += sum;
        }
    }
    const double* Di = &Dinv[(size_t)i * bb];
    for (int s = 0; s < cnt; ++s) {
      double* out = &P.vals[(size_t)(p0 + s) * pb];
      const double* tt = &T[(size_t)s * pb];
      for (int r = 0; r < bs; ++r)
        for (int c = 0; c < nb; ++c) {
          double sum = 0;
          for (int m = 0; m < bs; ++m) sum += Di[r * bs + m] * tt[m * nb + c];
          out[r * nb + c] = -omega * sum;
        }
      if (rowcols[i][s] == Lf.agg[i]) {
        const double* q = &Pt.vals[(size_t)i * pb];
        for (int t2 = 0; t2 < pb; ++t2) out[t2] += q[t2];
      }
    }
  }
  Lf.haveP = true;
  return true;
}

}  // namespace

// ================================================================= C ABI
extern "C" {

typedef struct Gen* egen_t;

// d = 2 or 3; ne elements per side; modulus_mode 0 (E = 1) or 1 (per-element lognormal(0,1), stream 4);
// dirichlet 1 (face ix = 0 clamped, R4) or 0 (Neumann operator for the invariant tests).
// order 1 (Q1) or 2 (Q2 elements, (2 ne + 1)^d nodes); agg_mode 0 (3^d node boxes) or 1 (seeded greedy covering).
egen_t egen_create2(int d, int ne, double nu, uint64_t seed, int modulus_mode, int dirichlet, int order, int agg_mode) {
  if ((d != 2 && d != 3) || ne < 1 || (order != 1 && order != 2) || (agg_mode != 0 && agg_mode != 1)) return nullptr;
  Gen* G = new Gen();
  G->d = d; G->ne = ne; G->nu = nu; G->seed = seed; G->modulus_mode = modulus_mode; G->dirichlet = dirichlet;
  G->order = order; G->agg_mode = agg_mode;
  G->levels.resize(1);
  build_fine_operator(*G);
  return G;
}
egen_t egen_create(int d, int ne, double nu, uint64_t seed, int modulus_mode, int dirichlet) {
  return egen_create2(d, ne, nu, seed, modulus_mode, dirichlet, 1, 0);
}
void egen_destroy(egen_t G) { delete G; }
const char* egen_error(egen_t G) { return G ? G->err.c_str() : "null handle"; }
int egen_nlevels(egen_t G) { return G ? (int)G->levels.size() : -1; }

// Borrow the arrays of a matrix.  which: 0 = A_level, 1 = P_level (level -> level+1), 2 = P_tent_level.
int egen_matrix(egen_t G, int level, int which, int32_t* nbrows, int32_t* nbcols, int32_t* bs_r, int32_t* bs_c,
                int64_t* nnzb, const int32_t** rowptr, const int32_t** colidx, const double** vals) {
  if (!G || level < 0 || level >= (int)G->levels.size()) return -1;
  Level& L = G->levels[level];
  const Bsr* M = nullptr;
  if (which == 0 && L.haveA) M = &L.A;
  if (which == 1 && L.haveP) M = &L.P;
  if (which == 2 && L.haveP) M = &L.Ptent;
  if (!M) return -2;
  *nbrows = M->nbrows; *nbcols = M->nbcols; *bs_r = M->bs_r; *bs_c = M->bs_c; *nnzb = M->nnzb();
  *rowptr = M->rowptr.data(); *colidx = M->colidx.data(); *vals = M->vals.data();
  return 0;
}

// Give the generator the operator of a coarse level (computed elsewhere: oracle in tests, the CUDA path in
// bench.py) so that the next prolongator can be built from it.  Arrays are copied.
int egen_set_operator(egen_t G, int level, int32_t nbrows, int32_t bs, int64_t nnzb, const int32_t* rowptr,
                      const int32_t* colidx, const double* vals) {
  if (!G || level < 1 || level >= (int)G->levels.size()) return -1;
  Level& L = G->levels[level];
  if (nbrows != L.nnodes() || bs != L.bs) return -3;
  L.A.nbrows = L.A.nbcols = nbrows; L.A.bs_r = L.A.bs_c = bs;
  L.A.rowptr.assign(rowptr, rowptr + nbrows + 1);
  L.A.colidx.assign(colidx, colidx + nnzb);
  L.A.vals.assign(vals, vals + nnzb * bs * bs);
  L.haveA = true;
  return 0;
}

// Build P_level (and the skeleton of level+1).  Returns 0 or a negative code; egen_error has the reason.
int egen_build_prolongator(egen_t G, int level) {
  if (!G || level < 0 || level >= (int)G->levels.size()) return -1;
  return build_P(*G, level) ? 0 : -4;
}

int egen_level_info(egen_t G, int level, int32_t* nnodes, int32_t* bs, int32_t* nb, int32_t nx[3], double* lambda,
                    double* omega) {
  if (!G || level < 0 || level >= (int)G->levels.size()) return -1;
  Level& L = G->levels[level];
  *nnodes = (int32_t)L.nnodes(); *bs = L.bs; *nb = L.nb;
  nx[0] = L.nx[0]; nx[1] = L.nx[1]; nx[2] = L.nx[2];
  *lambda = L.lambda; *omega = L.omega;
  return 0;
}

// coords: d per node; rfac: nb*nb per node (level >= 1, else null); agg: node -> aggregate (after build)
int egen_level_arrays(egen_t G, int level, const double** coords, const double** rfac, const int32_t** agg) {
  if (!G || level < 0 || level >= (int)G->levels.size()) return -1;
  Level& L = G->levels[level];
  *coords = L.coords.data();
  *rfac = L.Rfac.empty() ? nullptr : L.Rfac.data();
  *agg = L.agg.empty() ? nullptr : L.agg.data();
  return 0;
}

// reference element matrix (for pin I1): out has (d*(order+1)^d)^2 entries
int egen_element_matrix2(int d, int order, double h, double E, double nu, double* out) {
  if ((d != 2 && d != 3) || (order != 1 && order != 2)) return -1;
  std::vector<double> K;
  element_matrix(d, order, h, E, nu, K);
  std::memcpy(out, K.data(), sizeof(double) * K.size());
  return 0;
}
int egen_element_matrix(int d, double h, double E, double nu, double* out) {
  if (d != 2 && d != 3) return -1;
  std::vector<double> K;
  element_matrix(d, 1, h, E, nu, K);
  std::memcpy(out, K.data(), sizeof(double) * K.size());
  return 0;
}

// The finite-element contribution stream of elements [e0, e1) in ascending element order (blocked COO form,
// PAPER.md:248-250): per element (order+1)^(2d) (Q1: 16 / 64) contributions (a, b), a slowest; coordinate = (node of a, node
// of b); block = E_e * Ke[a][b] (d x d, row-major).  With Dirichlet the clamped face is folded into the stream: a
// block whose row or column node has ix = 0 is zero, except the node's own diagonal block, which carries
// I / (number of adjacent elements) so that the assembled block is exactly I (R4).  Any output may be null.
int egen_element_stream(egen_t G, int64_t e0, int64_t e1, int32_t* brow, int32_t* bcol, double* vals) {
  if (!G || e0 < 0 || e1 < e0) return -1;
  const int d = G->d, ne = G->ne, p = G->order, n1 = p + 1, n = p * ne + 1, bb = d * d;
  int nen = 1;
  for (int k = 0; k < d; ++k) nen *= n1;
  const int nd = d * nen;
  const int64_t NE = (int64_t)ne * ne * (d == 3 ? ne : 1);
  if (e1 > NE) return -2;
#pragma omp parallel for schedule(static)
  for (int64_t e = e0; e < e1; ++e) {
    const int ex = (int)(e % ne), ey = (int)((e / ne) % ne), ez = (d == 3) ? (int)(e / ((int64_t)ne * ne)) : 0;
    const double Ee = G->Emod.empty() ? 1.0 : G->Emod[(size_t)e];
    for (int a = 0; a < nen; ++a)
      for (int b = 0; b < nen; ++b) {
        const int64_t c = (e - e0) * nen * nen + a * nen + b;
        const int ax = p * ex + a % n1, ay = p * ey + (a / n1) % n1, az = (d == 3) ? p * ez + a / (n1 * n1) : 0;
        const int bx = p * ex + b % n1, by = p * ey + (b / n1) % n1, bz = (d == 3) ? p * ez + b / (n1 * n1) : 0;
        if (brow) brow[c] = (int32_t)(ax + (int64_t)n * (ay + (int64_t)n * az));
        if (bcol) bcol[c] = (int32_t)(bx + (int64_t)n * (by + (int64_t)n * bz));
        if (!vals) continue;
        double* blk = vals + (size_t)c * bb;
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) blk[i * d + j] = Ee * G->Ke[(size_t)(a * d + i) * nd + (b * d + j)];
        if (G->dirichlet && (ax == 0 || bx == 0)) {
          for (int t = 0; t < bb; ++t) blk[t] = 0.0;
          if (a == b) {   // number of elements that contain the node: 1 or 2 per transverse direction
            const int cy = el_hi(ay, p, ne) - el_lo(ay, p) + 1, cz = (d == 3) ? el_hi(az, p, ne) - el_lo(az, p) + 1 : 1;
            for (int i = 0; i < d; ++i) blk[i * d + i] = 1.0 / (double)(cy * cz);
          }
        }
      }
  }
  return 0;
}

// borrowed: per-element moduli (null when E = 1 everywhere) and the reference element matrix (E = 1)
int egen_element_data(egen_t G, const double** emod, const double** ke) {
  if (!G) return -1;
  *emod = G->Emod.empty() ? nullptr : G->Emod.data();
  *ke = G->Ke.data();
  return 0;
}

void egen_uniform(uint64_t seed, uint64_t purpose, int64_t n, double a, double b, double* out) {
  fill_uniform(seed, purpose, n, a, b, out);
}

}  // extern "C"
