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
  std::vector<Level> levels;
  std::vector<double> Emod;  // per-element modulus (empty: 1 everywhere)
  std::vector<double> Ke;    // reference element matrix (E = 1)
  std::string err;
};

// ---------------------------------------------------------------- O2: element matrix
// K[(a*d+i)][(b*d+j)] = int  lam d_i N_a d_j N_b + mu d_j N_a d_i N_b + mu delta_ij grad N_a . grad N_b
// Local node a has reference coordinates (+-1 per direction), bit k of a selects direction k (x fastest).
void element_matrix(int d, double h, double E, double nu, std::vector<double>& K) {
  const int nen = 1 << d, nd = d * nen;
  K.assign((size_t)nd * nd, 0.0);
  const double lam = E * nu / ((1 + nu) * (1 - 2 * nu)), mu = E / (2 * (1 + nu));
  const double g = 1.0 / std::sqrt(3.0);
  const double detJ = std::pow(h / 2, d);
  for (int q = 0; q < nen; ++q) {  // 2^d Gauss points, weight 1
    double xi[3] = {0, 0, 0};
    for (int k = 0; k < d; ++k) xi[k] = ((q >> k) & 1) ? g : -g;
    double dN[8][3];
    for (int a = 0; a < nen; ++a)
      for (int k = 0; k < d; ++k) {
        double v = 1;
        for (int m = 0; m < d; ++m) {
          double s = ((a >> m) & 1) ? 1.0 : -1.0;
          v *= (m == k) ? s / 2 : (1 + s * xi[m]) / 2;
        }
        dN[a][k] = v * (2 / h);
      }
    for (int a = 0; a < nen; ++a)
      for (int b = 0; b < nen; ++b) {
        double gg = 0;
        for (int k = 0; k < d; ++k) gg += dN[a][k] * dN[b][k];
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) {
            double v = lam * dN[a][i] * dN[b][j] + mu * dN[a][j] * dN[b][i] + (i == j ? mu * gg : 0.0);
            K[(size_t)(a * d + i) * nd + (b * d + j)] += v * detJ;
          }
      }
  }
}

// ---------------------------------------------------------------- O1, O3, O4: fine operator
inline int clip_lo(int i) { return i > 0 ? -1 : 0; }
inline int clip_hi(int i, int n) { return i < n - 1 ? 1 : 0; }

void build_fine_operator(Gen& G) {
  Level& L = G.levels[0];
  const int d = G.d, n = G.ne + 1, ne = G.ne;
  L.d = d; L.bs = d; L.nb = (d == 3) ? 6 : 3;
  L.nx[0] = n; L.nx[1] = n; L.nx[2] = (d == 3) ? n : 1;
  const int nz = L.nx[2];
  const int64_t N = L.nnodes();
  const double h = 1.0 / ne;
  L.coords.resize((size_t)N * d);
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        int64_t id = ix + (int64_t)n * (iy + (int64_t)n * iz);
        L.coords[id * d + 0] = ix * h;
        L.coords[id * d + 1] = iy * h;
        if (d == 3) L.coords[id * d + 2] = iz * h;
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
  element_matrix(d, h, 1.0, G.nu, Ke);
  const int nen = 1 << d, nd = d * nen, bb = d * d;

  Bsr& A = L.A;
  A.nbrows = A.nbcols = (int32_t)N; A.bs_r = A.bs_c = d;
  A.rowptr.assign(N + 1, 0);
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        int64_t id = ix + (int64_t)n * (iy + (int64_t)n * iz);
        int cx = clip_hi(ix, n) - clip_lo(ix) + 1, cy = clip_hi(iy, n) - clip_lo(iy) + 1;
        int cz = (d == 3) ? clip_hi(iz, nz) - clip_lo(iz) + 1 : 1;
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
        const int lx = clip_lo(ix), ly = clip_lo(iy), lz = (d == 3) ? clip_lo(iz) : 0;
        const int cx = clip_hi(ix, n) - lx + 1, cy = clip_hi(iy, n) - ly + 1;
        const int cz = (d == 3) ? clip_hi(iz, nz) - lz + 1 : 1;
        const int64_t base = A.rowptr[id];
        for (int sz = 0; sz < cz; ++sz)
          for (int sy = 0; sy < cy; ++sy)
            for (int sx = 0; sx < cx; ++sx)
              A.colidx[base + (sz * cy + sy) * cx + sx] =
                  (int32_t)((ix + lx + sx) + (int64_t)n * ((iy + ly + sy) + (int64_t)n * (iz + lz + sz)));
        // gather form of the element loop: adjacent elements in ascending element id
        for (int oz = (d == 3 ? -1 : 0); oz <= 0; ++oz)
          for (int oy = -1; oy <= 0; ++oy)
            for (int ox = -1; ox <= 0; ++ox) {
              const int ex = ix + ox, ey = iy + oy, ez = iz + oz;
              if (ex < 0 || ex >= ne || ey < 0 || ey >= ne) continue;
              if (d == 3 && (ez < 0 || ez >= ne)) continue;
              const int64_t e = ex + (int64_t)ne * (ey + (int64_t)ne * (d == 3 ? ez : 0));
              const double Ee = Emod.empty() ? 1.0 : Emod[e];
              const int a = (-ox) | ((-oy) << 1) | ((d == 3 ? -oz : 0) << 2);
              for (int b = 0; b < nen; ++b) {
                const int dx = ox + (b & 1), dy = oy + ((b >> 1) & 1), dz = (d == 3) ? oz + ((b >> 2) & 1) : 0;
                const int64_t slot = base + ((dz - lz) * cy + (dy - ly)) * cx + (dx - lx);
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
  for (int k = 0; k < d; ++k) na[k] = std::max(1, L.nx[k] / 3);
  const int64_t NA = (int64_t)na[0] * na[1] * na[2];
  L.agg.resize(N);
  std::vector<std::vector<int32_t>> members(NA);
  for (int iz = 0; iz < L.nx[2]; ++iz)
    for (int iy = 0; iy < L.nx[1]; ++iy)
      for (int ix = 0; ix < L.nx[0]; ++ix) {
        const int64_t id = ix + (int64_t)L.nx[0] * (iy + (int64_t)L.nx[1] * iz);
        const int ax = std::min(ix / 3, na[0] - 1), ay = std::min(iy / 3, na[1] - 1);
        const int az = (d == 3) ? std::min(iz / 3, na[2] - 1) : 0;
        const int64_t J = ax + (int64_t)na[0] * (ay + (int64_t)na[1] * az);
        L.agg[id] = (int32_t)J;
        members[J].push_back((int32_t)id);  // ascending node id
      }
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
egen_t egen_create(int d, int ne, double nu, uint64_t seed, int modulus_mode, int dirichlet) {
  if ((d != 2 && d != 3) || ne < 1) return nullptr;
  Gen* G = new Gen();
  G->d = d; G->ne = ne; G->nu = nu; G->seed = seed; G->modulus_mode = modulus_mode; G->dirichlet = dirichlet;
  G->levels.resize(1);
  build_fine_operator(*G);
  return G;
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

// reference element matrix (for pin I1): out has (d*2^d)^2 entries
int egen_element_matrix(int d, double h, double E, double nu, double* out) {
  if (d != 2 && d != 3) return -1;
  std::vector<double> K;
  element_matrix(d, h, E, nu, K);
  std::memcpy(out, K.data(), sizeof(double) * K.size());
  return 0;
}

// The finite-element contribution stream of elements [e0, e1) in ascending element order (blocked COO form,
// PAPER.md:248-250): per element 4^d (2D: 16, 3D: 64) contributions (a, b), a slowest; coordinate = (node of a, node
// of b); block = E_e * Ke[a][b] (d x d, row-major).  With Dirichlet the clamped face is folded into the stream: a
// block whose row or column node has ix = 0 is zero, except the node's own diagonal block, which carries
// I / (number of adjacent elements) so that the assembled block is exactly I (R4).  Any output may be null.
int egen_element_stream(egen_t G, int64_t e0, int64_t e1, int32_t* brow, int32_t* bcol, double* vals) {
  if (!G || e0 < 0 || e1 < e0) return -1;
  const int d = G->d, ne = G->ne, n = ne + 1, nen = 1 << d, nd = d * nen, bb = d * d;
  const int64_t NE = (int64_t)ne * ne * (d == 3 ? ne : 1);
  if (e1 > NE) return -2;
#pragma omp parallel for schedule(static)
  for (int64_t e = e0; e < e1; ++e) {
    const int ex = (int)(e % ne), ey = (int)((e / ne) % ne), ez = (d == 3) ? (int)(e / ((int64_t)ne * ne)) : 0;
    const double Ee = G->Emod.empty() ? 1.0 : G->Emod[(size_t)e];
    for (int a = 0; a < nen; ++a)
      for (int b = 0; b < nen; ++b) {
        const int64_t c = (e - e0) * nen * nen + a * nen + b;
        const int ax = ex + (a & 1), ay = ey + ((a >> 1) & 1), az = ez + ((a >> 2) & 1);
        const int bx = ex + (b & 1), by = ey + ((b >> 1) & 1), bz = ez + ((b >> 2) & 1);
        if (brow) brow[c] = (int32_t)(ax + (int64_t)n * (ay + (int64_t)n * az));
        if (bcol) bcol[c] = (int32_t)(bx + (int64_t)n * (by + (int64_t)n * bz));
        if (!vals) continue;
        double* blk = vals + (size_t)c * bb;
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) blk[i * d + j] = Ee * G->Ke[(size_t)(a * d + i) * nd + (b * d + j)];
        if (G->dirichlet && (ax == 0 || bx == 0)) {
          for (int t = 0; t < bb; ++t) blk[t] = 0.0;
          if (a == b) {
            const int cy = (ay > 0 && ay < ne) ? 2 : 1, cz = (d == 3 && az > 0 && az < ne) ? 2 : 1;
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
