// vcycle.cu -- V-cycle over the reused hierarchy, polynomial point-block-Jacobi smoother, dense coarsest solve, PCG.
//
// PAPER.md:42 (two-level cycle: pre-smooth, form and restrict the residual, coarse correction, prolong and add,
// post-smooth; recursion gives the V-cycle); 83, 121 (the V-cycle is the recurring, SpMV-bound solve phase);
// 113 (point-block Jacobi smoother, CG accelerator, unpreconditioned residual norm).
// The smoother is the Chebyshev polynomial in D^-1 A named by BASELINE.json config 4 (reading R15):
//   theta=(lmax+lmin)/2, delta=(lmax-lmin)/2, sigma=theta/delta, rho_0=1/sigma
//   r=b-Ax; d_0=D^-1 r/theta; x+=d_0;
//   k=1..deg-1: r-=A d_{k-1}; rho_k=1/(2 sigma-rho_{k-1}); d_k=rho_k rho_{k-1} d_{k-1}+(2 rho_k/delta) D^-1 r; x+=d_k
// Every SpMV runs in the blocked kernels of bsr.cu with the vector update fused into its epilogue
// (r = b - A x, r -= A d, x += P e); D^-1 r and the d/x update are one small kernel.
// Coarsest level (reading R17): dense Cholesky A = L L^T on the device -- right-looking with 128-wide panels
// (32x32 tile kernels inside a panel, ONE register-tiled fp64 GEMM, dense_gemm.cu, for every trailing update) -- then
// the explicit triangular inverse L^-1 by recursive doubling (X21 = -X22 (L21 X11), two batched GEMMs per level), so
// that every later solve is two fully parallel triangular mat-vecs.
#include <algorithm>
#include <cmath>

#include "internal.h"

namespace bsramg {

constexpr int TS = 32;  // tile size of the dense coarsest-level kernels

struct Level {
  bsr_t A = nullptr, P = nullptr;
  double lambda = 0;
  int64_t n = 0;
  int bs = 0;
  double *Dinv = nullptr, *r = nullptr, *t = nullptr, *d = nullptr, *b = nullptr, *x = nullptr;   // t = A * (x or d)
};

}  // namespace bsramg

struct vcycle_s {
  uint64_t magic = 0;
  int nlevels = 0, degree = 2;
  double lo = 0.1, hi = 1.1;
  std::vector<bsramg::Level> L;
  // coarsest level, dense
  int64_t nc = 0, npad = 0;
  int64_t band = 0;   // scalar half-bandwidth of the coarsest operator, rounded up to whole panels (npad: not banded)
  double *dense = nullptr, *linv = nullptr, *linvT = nullptr, *ytmp = nullptr;
  int32_t* coarse_rowidx = nullptr;   // block row of every stored block of the coarsest operator (dense fill)
  int* d_status = nullptr;
  // PCG work space
  double *pr = nullptr, *pz = nullptr, *pp = nullptr, *pq = nullptr, *partial = nullptr, *scal = nullptr;
};
static const uint64_t VC_MAGIC = 0x5643594330303031ull;

namespace bsramg {

// ------------------------------------------------------------------ point-block Jacobi data: D^-1 per block row
template <int BS>
__global__ void __launch_bounds__(128)
dinv_kernel(int32_t nbrows, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
            const double* __restrict__ vals, double* __restrict__ dinv, int* __restrict__ status) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nbrows) return;
  int32_t kd = -1;
  for (int32_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
    if (colidx[k] == i) { kd = k; break; }
  double M[BS][2 * BS];
#pragma unroll
  for (int r = 0; r < BS; ++r)
#pragma unroll
    for (int c = 0; c < BS; ++c) {
      M[r][c] = (kd >= 0) ? vals[(int64_t)kd * BS * BS + r * BS + c] : 0.0;
      M[r][BS + c] = (r == c) ? 1.0 : 0.0;
    }
  bool ok = kd >= 0;
  // Gauss-Jordan with partial pivoting, fully unrolled (row swaps by value exchange)
#pragma unroll
  for (int c = 0; c < BS; ++c) {
#pragma unroll
    for (int r = c + 1; r < BS; ++r) {
      if (fabs(M[r][c]) > fabs(M[c][c])) {
#pragma unroll
        for (int j = 0; j < 2 * BS; ++j) { const double t = M[r][j]; M[r][j] = M[c][j]; M[c][j] = t; }
      }
    }
    const double piv = M[c][c];
    if (piv == 0.0) ok = false;
    const double ip = 1.0 / piv;
#pragma unroll
    for (int j = 0; j < 2 * BS; ++j) M[c][j] *= ip;
#pragma unroll
    for (int r = 0; r < BS; ++r) {
      if (r != c) {
        const double f = M[r][c];
#pragma unroll
        for (int j = 0; j < 2 * BS; ++j) M[r][j] = fma(-f, M[c][j], M[r][j]);
      }
    }
  }
  if (!ok) atomicOr(status, 1);
#pragma unroll
  for (int r = 0; r < BS; ++r)
#pragma unroll
    for (int c = 0; c < BS; ++c) dinv[(int64_t)i * BS * BS + r * BS + c] = M[r][BS + c];
}

// One Chebyshev step on the residual r = base - t, where t = A*(x or d) is the plain SpMV's output (t == nullptr: r is
// `base` itself).  The subtraction the fused-epilogue SpMVs r = b - A x / r -= A d did per row (at +10 % over the plain
// y = A x, bsr.cu) happens here, on vectors this kernel streams anyway; the results are bit-identical.
//   z = D^-1 r (block row wise);  d = cd*d + cz*z  (first step: d = z/theta);  x = d or x += d;
//   r_out (may alias base), when a later step needs r.   One thread per block row.
template <int BS>
__global__ void __launch_bounds__(256)
cheb_update_kernel(int64_t nb, const double* __restrict__ dinv, const double* base, const double* __restrict__ t,
                   double* r_out, double* __restrict__ d, double* __restrict__ x, int first, double theta, double cd,
                   double cz, int x_zero) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nb) return;
  double r[BS];
#pragma unroll
  for (int b = 0; b < BS; ++b) r[b] = t ? base[i * BS + b] - t[i * BS + b] : base[i * BS + b];
#pragma unroll
  for (int a = 0; a < BS; ++a) {
    double z = 0.0;
#pragma unroll
    for (int b = 0; b < BS; ++b) z = fma(dinv[(i * BS + a) * BS + b], r[b], z);
    const int64_t e = i * BS + a;
    const double dn = first ? z / theta : cd * d[e] + cz * z;
    d[e] = dn;
    x[e] = x_zero ? dn : x[e] + dn;
    if (r_out) r_out[e] = r[a];
  }
}

int block_diag_inverse(bsr_t A, double* dinv, int* status, cudaStream_t st) {
  const unsigned grid = (unsigned)((A->nbrows + 127) / 128);
  if (!grid) return BSR_OK;
  switch (A->bs_r) {
    case 2: LAUNCH(dinv_kernel<2>, grid, 128, 0, st, A->nbrows, A->d_rowptr, A->d_colidx, A->d_vals, dinv, status); break;
    case 3: LAUNCH(dinv_kernel<3>, grid, 128, 0, st, A->nbrows, A->d_rowptr, A->d_colidx, A->d_vals, dinv, status); break;
    case 6: LAUNCH(dinv_kernel<6>, grid, 128, 0, st, A->nbrows, A->d_rowptr, A->d_colidx, A->d_vals, dinv, status); break;
    default: return fail(BSR_ERR_BLOCK, "unsupported block size %d", A->bs_r);
  }
  return BSR_OK;
}

static int launch_dinv(Level& lv, int* status, cudaStream_t st) { return block_diag_inverse(lv.A, lv.Dinv, status, st); }

// r = b - t, two entries per thread (one 16-byte access each when the three vectors are 16-byte aligned)
__global__ void __launch_bounds__(256)
resid_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ t, double* __restrict__ r) {
  const int64_t e = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 2;
  const bool aligned = ((reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(t) | reinterpret_cast<uintptr_t>(r)) & 15) == 0;
  if (e + 1 < n && !aligned) {
    r[e] = b[e] - t[e];
    r[e + 1] = b[e + 1] - t[e + 1];
  } else if (e + 1 < n) {
    const double2 bv = *reinterpret_cast<const double2*>(b + e), tv = *reinterpret_cast<const double2*>(t + e);
    *reinterpret_cast<double2*>(r + e) = make_double2(bv.x - tv.x, bv.y - tv.y);
  } else if (e < n) {
    r[e] = b[e] - t[e];
  }
}

static int launch_cheb(Level& lv, double* x, const double* base, const double* t, double* r_out, int first, double theta,
                       double cd, double cz, int x_zero, cudaStream_t st) {
  const int64_t nb = lv.n / lv.bs;
  const unsigned grid = (unsigned)((nb + 255) / 256);
  if (!grid) return BSR_OK;
  switch (lv.bs) {
    case 2: LAUNCH(cheb_update_kernel<2>, grid, 256, 0, st, nb, lv.Dinv, base, t, r_out, lv.d, x, first, theta, cd, cz, x_zero); break;
    case 3: LAUNCH(cheb_update_kernel<3>, grid, 256, 0, st, nb, lv.Dinv, base, t, r_out, lv.d, x, first, theta, cd, cz, x_zero); break;
    case 6: LAUNCH(cheb_update_kernel<6>, grid, 256, 0, st, nb, lv.Dinv, base, t, r_out, lv.d, x, first, theta, cd, cz, x_zero); break;
    default: return fail(BSR_ERR_BLOCK, "unsupported block size %d", lv.bs);
  }
  return BSR_OK;
}

// one polynomial smoother application on level l: x <- x + p(D^-1 A)(b - A x); x_zero: x is known to be 0.
// The residual of step k is kept as the pair (base, t): r_0 = b - A x (r_0 = b exactly from the zero guess),
// r_k = r_{k-1} - A d_{k-1}; it is written out (lv.r) only when a later step reads it.
static int smooth(vcycle_t vc, int l, const double* b, double* x, bool x_zero, cudaStream_t st) {
  Level& lv = vc->L[l];
  const double lmin = vc->lo * lv.lambda, lmax = vc->hi * lv.lambda;
  const double theta = (lmax + lmin) / 2, delta = (lmax - lmin) / 2, sigma = theta / delta;
  const double* base = b;
  double rho = 1 / sigma;
  for (int k = 0; k < vc->degree; ++k) {
    const double* t = nullptr;
    if (k == 0 && !x_zero) { BSR_TRY(spmv_launch(lv.A, x, lv.t, nullptr, EPI_ASSIGN, st)); t = lv.t; }     // r_0 = b - A x
    if (k > 0) { BSR_TRY(spmv_launch(lv.A, lv.d, lv.t, nullptr, EPI_ASSIGN, st)); t = lv.t; }             // r_k = r_{k-1} - A d_{k-1}
    // from the zero guess x = d_0, so r_1 = b - A d_0 needs no stored r_0
    double* r_out = (t && k + 1 < vc->degree) ? lv.r : nullptr;
    if (k == 0) {
      BSR_TRY(launch_cheb(lv, x, base, t, r_out, 1, theta, 0.0, 0.0, x_zero ? 1 : 0, st));
    } else {
      const double rho_new = 1 / (2 * sigma - rho);
      BSR_TRY(launch_cheb(lv, x, base, t, r_out, 0, theta, rho_new * rho, 2 * rho_new / delta, 0, st));
      rho = rho_new;
    }
    if (r_out) base = lv.r;
  }
  return BSR_OK;
}

// ------------------------------------------------------------------ coarsest level: dense Cholesky + L^-1
// dense is npad x npad row-major, npad a multiple of TS; rows/cols >= nc carry the identity.
// zero row i of an npad x npad matrix from `reach` columns left of its diagonal 128-block to the end of that block: the
// part of the matrix the banded factorisation reads and writes
__global__ void __launch_bounds__(256)
band_zero_kernel(int64_t npad, int64_t reach, double* __restrict__ mat) {
  const int64_t i = blockIdx.x, blk0 = (i / 128) * 128;
  const int64_t c0 = blk0 > reach ? blk0 - reach : 0, c1 = blk0 + 128;
  double2* row = reinterpret_cast<double2*>(mat + i * npad);
  for (int64_t c = c0 / 2 + threadIdx.x; c < c1 / 2; c += blockDim.x) row[c] = make_double2(0.0, 0.0);
}

__global__ void dense_pad_kernel(int64_t nc, int64_t npad, double* __restrict__ dense) {
  const int64_t i = nc + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < npad) dense[i * npad + i] = 1.0;
}

__global__ void __launch_bounds__(256)
dense_fill_kernel(int64_t nvals, int bs, const int32_t* __restrict__ rowidx_of_slot, const int32_t* __restrict__ colidx,
                  const double* __restrict__ vals, int64_t npad, double* __restrict__ dense) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nvals) return;
  const int bb = bs * bs;
  const int64_t k = e / bb;
  const int pos = (int)(e - k * bb);
  const int r = pos / bs, c = pos - r * bs;
  dense[((int64_t)rowidx_of_slot[k] * bs + r) * npad + (int64_t)colidx[k] * bs + c] = vals[e];
}

// ---- the diagonal 128-block of a panel: Cholesky factor AND inverse in one CTA, all in shared memory.
// The block lives as its ten lower 32x32 tiles (rows padded to PL doubles).  Per tile column s: one warp factors the
// diagonal tile out of registers (below), then the tiles under it are solved (L_is = A_is X_ss^T) and the rest of the
// block updated (A_ik -= L_is L_ks^T) on the fp64 tensor-core path, a 32x32 tile product shared by four warps (a 16x16
// quadrant = 2x2 mma.sync m8n8k4 fragments each).  The inverse follows by the tile recurrence
//   X_ij = -X_ii * sum_{k=j}^{i-1} L_ik X_kj   (i > j, one sub-diagonal after the other).
constexpr int PANEL = 128, PT = PANEL / TS;
constexpr int PL = 36;                                  // padded tile row: fragment loads hit 16 distinct banks
constexpr int PTILES = PT * (PT + 1) / 2;
constexpr int PANEL_SMEM = 2 * PTILES * TS * PL * 8;    // L tiles + X tiles: 184,320 bytes
__device__ __forceinline__ int ltile(int i, int j) { return (i * (i + 1) / 2 + j) * TS * PL; }

// The 32 steps of a tile are a dependent chain (pivot -> 1/sqrt -> column -> update of the next pivot), so ONE warp runs
// them with no barrier: lane r holds row r of the tile and COLUMN r of X = L^-1 (forward substitution of the identity
// with each column of L as soon as it is final), so that the value both updates need in step k, l_i = L[i][k], comes
// from the same shuffle:
//   a[r][i] -= l_r l_i  (k < i <= r)        X[i][c] -= l_i X[k][c]  (c <= k < i, lane c)
// Both run unpredicated: l_r is 0 for r <= k, X[k][c] is still exactly 0 for c > k, and what lands above the diagonal
// of a row is never read.  The pivot's reciprocal square root (rsqrt, <= 1 ulp) replaces sqrt followed by divisions on
// the critical path; L[k][k] itself is p * rsqrt(p).
__device__ __forceinline__ void potrf_warp(double* __restrict__ a, double* __restrict__ x, int r, int* status) {
  double ar[TS], xc[TS];
#pragma unroll
  for (int c = 0; c < TS; ++c) { ar[c] = a[r * PL + c]; xc[c] = (c == r) ? 1.0 : 0.0; }
  __syncwarp();
  bool bad = false;
#pragma unroll
  for (int k = 0; k < TS; ++k) {
    double p = __shfl_sync(0xffffffffu, ar[k], k);
    if (!(p > 0.0)) { bad = true; p = 1.0; }
    const double rd = rsqrt(p);
    const double l = (r > k) ? ar[k] * rd : 0.0;             // L[r][k] below the diagonal
    ar[k] = (r == k) ? p * rd : l;
    xc[k] *= rd;                                              // row k of X (zero right of the diagonal)
    const double xk = xc[k];
#pragma unroll
    for (int i = k + 1; i < TS; ++i) {
      const double li = __shfl_sync(0xffffffffu, l, i);
      ar[i] = fma(-l, li, ar[i]);
      xc[i] = fma(-li, xk, xc[i]);
    }
  }
  if (bad && r == 0) atomicOr(status, 2);
#pragma unroll
  for (int c = 0; c < TS; ++c) {
    a[r * PL + c] = (c <= r) ? ar[c] : 0.0;
    x[c * PL + r] = (c >= r) ? xc[c] : 0.0;                   // X[c][r]
  }
}

// acc += A[qm.., :] * op(B)[:, qn..] over the 32 k of a tile; op(B)[k][n] = B[n][k] when TB (B given as n x k)
template <bool TB>
__device__ __forceinline__ void quad_mma(double (&acc)[2][2][2], const double* __restrict__ A,
                                         const double* __restrict__ B, int qm, int qn, int lane) {
  const int fk = lane & 3, fr = lane >> 2;
#pragma unroll
  for (int k0 = 0; k0 < TS; k0 += 4) {
    double af[2], bf[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) af[i] = A[(qm + 8 * i + fr) * PL + k0 + fk];
#pragma unroll
    for (int j = 0; j < 2; ++j) bf[j] = TB ? B[(qn + 8 * j + fr) * PL + k0 + fk] : B[(k0 + fk) * PL + qn + 8 * j + fr];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(af[i]), "d"(bf[j]));
  }
}

// C[quadrant] = beta * C + alpha * acc
__device__ __forceinline__ void quad_store(double* __restrict__ C, const double (&acc)[2][2][2], int qm, int qn, int lane,
                                           double alpha, double beta) {
  const int fk = lane & 3, fr = lane >> 2;
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      double2* cp = reinterpret_cast<double2*>(C + (qm + 8 * i + fr) * PL + qn + 8 * j + 2 * fk);
      double2 v = make_double2(alpha * acc[i][j][0], alpha * acc[i][j][1]);
      if (beta != 0.0) { const double2 o = *cp; v.x = fma(beta, o.x, v.x); v.y = fma(beta, o.y, v.y); }
      *cp = v;
    }
}

__global__ void __launch_bounds__(256)
potrf_panel_kernel(int64_t npad, int J, double* __restrict__ dense, double* __restrict__ linv, int* __restrict__ status) {
  extern __shared__ __align__(16) double panel_sm[];
  double* Lt = panel_sm;
  double* Xt = panel_sm + PTILES * TS * PL;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int group = warp >> 2, qm = ((warp >> 1) & 1) * 16, qn = (warp & 1) * 16;   // two groups of four warps
  double* blk = dense + ((int64_t)J * PANEL) * npad + (int64_t)J * PANEL;
  double* xblk = linv + ((int64_t)J * PANEL) * npad + (int64_t)J * PANEL;
  // 16-byte accesses: PL is even and npad a multiple of 128, so every tile row starts on 16 bytes on both sides
#pragma unroll 4
  for (int e = tid; e < PTILES * TS * TS / 2; e += 256) {
    const int tl = e >> 9, r = (e >> 4) & 31, c = (e & 15) * 2;
    const int ti = (tl >= 6) ? 3 : (tl >= 3) ? 2 : (tl >= 1) ? 1 : 0, tj = tl - ti * (ti + 1) / 2;
    *reinterpret_cast<double2*>(Lt + tl * TS * PL + r * PL + c) =
        *reinterpret_cast<const double2*>(blk + (int64_t)(ti * TS + r) * npad + tj * TS + c);
  }
  __syncthreads();
  for (int s = 0; s < PT; ++s) {
    if (warp == 0) potrf_warp(Lt + ltile(s, s), Xt + ltile(s, s), lane, status);
    __syncthreads();
    const int nt = PT - 1 - s;
    for (int j0 = 0; j0 < nt; j0 += 2) {                       // tiles below: L_is = A_is X_ss^T
      const int i = s + 1 + j0 + group;
      const bool on = j0 + group < nt;
      double acc[2][2][2] = {};
      if (on) quad_mma<true>(acc, Lt + ltile(i, s), Xt + ltile(s, s), qm, qn, lane);
      __syncthreads();                                         // every quadrant has read the tile it is about to overwrite
      if (on) quad_store(Lt + ltile(i, s), acc, qm, qn, lane, 1.0, 0.0);
    }
    __syncthreads();
    const int njobs = nt * (nt + 1) / 2;                       // A_ik -= L_is L_ks^T, s < k <= i
    for (int job = group; job < njobs; job += 2) {
      const int di = (job >= 3) ? 2 : (job >= 1) ? 1 : 0, dk = job - di * (di + 1) / 2;
      const int i = s + 1 + di, k = s + 1 + dk;
      double acc[2][2][2] = {};
      quad_mma<true>(acc, Lt + ltile(i, s), Lt + ltile(k, s), qm, qn, lane);
      quad_store(Lt + ltile(i, k), acc, qm, qn, lane, -1.0, 1.0);
    }
    __syncthreads();
  }
  for (int d = 1; d < PT; ++d) {                               // X, one sub-diagonal of tiles after the other
    const int nj = PT - d;
    for (int j0 = 0; j0 < nj; j0 += 2) {
      const int j = j0 + group, i = j + d;
      const bool on = j < nj;
      double acc[2][2][2] = {};
      if (on) {
        for (int k = j; k < i; ++k) quad_mma<false>(acc, Lt + ltile(i, k), Xt + ltile(k, j), qm, qn, lane);
        quad_store(Xt + ltile(i, j), acc, qm, qn, lane, 1.0, 0.0);   // T = sum_k L_ik X_kj, staged in X_ij's place
      }
      __syncthreads();
      double acc2[2][2][2] = {};
      if (on) quad_mma<false>(acc2, Xt + ltile(i, i), Xt + ltile(i, j), qm, qn, lane);
      __syncthreads();
      if (on) quad_store(Xt + ltile(i, j), acc2, qm, qn, lane, -1.0, 0.0);
      __syncthreads();
    }
  }
#pragma unroll 4
  for (int e = tid; e < PTILES * TS * TS / 2; e += 256) {
    const int tl = e >> 9, r = (e >> 4) & 31, c = (e & 15) * 2;
    const int ti = (tl >= 6) ? 3 : (tl >= 3) ? 2 : (tl >= 1) ? 1 : 0, tj = tl - ti * (ti + 1) / 2;
    const int64_t g = (int64_t)(ti * TS + r) * npad + tj * TS + c;
    *reinterpret_cast<double2*>(blk + g) = *reinterpret_cast<const double2*>(Lt + tl * TS * PL + r * PL + c);
    *reinterpret_cast<double2*>(xblk + g) = *reinterpret_cast<const double2*>(Xt + tl * TS * PL + r * PL + c);
  }
}

__global__ void __launch_bounds__(TS * TS)
transpose_tile_kernel(int64_t npad, const double* __restrict__ src, double* __restrict__ dst) {
  __shared__ double t[TS][TS + 1];
  const int tx = threadIdx.x, ty = threadIdx.y;
  if (blockIdx.x > blockIdx.y) return;   // src is lower triangular: its upper tiles are zero and dst's lower tiles are never read
  t[ty][tx] = src[((int64_t)blockIdx.y * TS + ty) * npad + (int64_t)blockIdx.x * TS + tx];
  __syncthreads();
  dst[((int64_t)blockIdx.x * TS + ty) * npad + (int64_t)blockIdx.y * TS + tx] = t[tx][ty];
}

// y[i] = sum_{j in [j0(i), j1(i))} M[i][j] x[j]; lower: j in [0, i]; upper: j in [i, n).  One CTA of 8 warps per row
// (a single warp streaming a 48 KB row has 2 KB in flight per memory latency: the long rows alone took 24 us),
// 16-byte loads, four of them in flight per thread on four partial sums; warp sums, then the 8 warps in order: a
// fixed summation tree, deterministic.
constexpr int TRIGEMV_THREADS = 256;
__global__ void __launch_bounds__(TRIGEMV_THREADS)
trigemv_kernel(int64_t n, int64_t npad, const double* __restrict__ M, const double* __restrict__ x,
               double* __restrict__ y, int upper) {
  __shared__ double wsum[TRIGEMV_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t i = blockIdx.x;
  const double* row = M + i * npad;                                  // 16-byte aligned (npad is a multiple of 128)
  const int64_t j0 = upper ? (i & ~31LL) : 0, j1 = upper ? n : i + 1;  // M is 0 outside the triangle; j0 is even
  double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
  if ((reinterpret_cast<uintptr_t>(x) & 15) == 0) {
    const double2* r2 = reinterpret_cast<const double2*>(row);
    const double2* x2 = reinterpret_cast<const double2*>(x);
    const int64_t p1 = j1 >> 1;                                      // whole pairs [j0/2, p1)
    for (int64_t p = (j0 >> 1) + tid; p < p1; p += 4 * TRIGEMV_THREADS) {
      double2 m[4], v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int64_t q = min(p + TRIGEMV_THREADS * u, p1 - 1);      // clamped: a repeated pair is weighted 0 below
        m[u] = __ldcs(r2 + q);
        v[u] = __ldg(x2 + q);
      }
      if (p + TRIGEMV_THREADS >= p1) m[1] = make_double2(0.0, 0.0);
      if (p + 2 * TRIGEMV_THREADS >= p1) m[2] = make_double2(0.0, 0.0);
      if (p + 3 * TRIGEMV_THREADS >= p1) m[3] = make_double2(0.0, 0.0);
      s0 = fma(m[0].y, v[0].y, fma(m[0].x, v[0].x, s0));
      s1 = fma(m[1].y, v[1].y, fma(m[1].x, v[1].x, s1));
      s2 = fma(m[2].y, v[2].y, fma(m[2].x, v[2].x, s2));
      s3 = fma(m[3].y, v[3].y, fma(m[3].x, v[3].x, s3));
    }
    if ((j1 & 1) && tid == 0) s0 = fma(row[j1 - 1], x[j1 - 1], s0);   // the odd last entry
  } else {
    for (int64_t j = j0 + tid; j < j1; j += TRIGEMV_THREADS) s0 = fma(row[j], x[j], s0);
  }
  double s = (s0 + s1) + (s2 + s3);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) wsum[warp] = s;
  __syncthreads();
  if (tid == 0) {
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < TRIGEMV_THREADS / 32; ++w) tot += wsum[w];
    y[i] = tot;
  }
}

static int coarse_factor(vcycle_t vc, cudaStream_t st) {
  bsr_t A = vc->L[vc->nlevels - 1].A;
  const int64_t np = vc->npad;            // a multiple of PANEL
  const int nb = (int)(np / TS), npan = (int)(np / PANEL);
  // what the banded factorisation touches is cleared, nothing else: in `dense` the band below and the 128-block on the
  // diagonal (fill-in and the inverse's workspace of the last refresh); in linvT, which holds L's panels until the final
  // transpose, the band plus the two tile rows by which the k-ranges of the inverse overshoot it.  linv is written in
  // its lower part only and was cleared once, at creation.
  const int64_t band0 = std::min(vc->band, np);
  LAUNCH(band_zero_kernel, (unsigned)np, 256, 0, st, np, band0, vc->dense);
  LAUNCH(band_zero_kernel, (unsigned)np, 256, 0, st, np, band0 + 256, vc->linvT);
  if (np > vc->nc) LAUNCH(dense_pad_kernel, (unsigned)((np - vc->nc + 63) / 64), 64, 0, st, vc->nc, np, vc->dense);
  const int64_t nvals = A->nnzb * A->bs_r * A->bs_c;
  if (nvals)
    LAUNCH(dense_fill_kernel, (unsigned)((nvals + 255) / 256), 256, 0, st, nvals, (int)A->bs_r, vc->coarse_rowidx,
           A->d_colidx, A->d_vals, np, vc->dense);
  const dim3 tb(TS, TS);
  // ---- A = L L^T, right-looking over 128-wide panels: the diagonal block (factor + inverse, one CTA), the panel below
  // it L21 = A21 X11^T and the trailing update, both GEMMs.  L21 is written OUT of place, into linvT (the GEMM's tiles
  // would otherwise overwrite what their neighbours still read): from here to the final transpose linvT holds the
  // off-diagonal panels of L and the strictly lower part of `dense` is free -- the workspace of the inverse below.
  // A banded operator (the lexicographic 27-point coarse grid: half-bandwidth 666 of 6000) keeps its band in L: below
  // the band every tile is zero and is skipped -- rows of a panel, of the trailing update and k-ranges of the inverse
  const int64_t band = std::min(vc->band, np);
  for (int J = 0; J < npan; ++J) {
    LAUNCH(potrf_panel_kernel, 1, 256, PANEL_SMEM, st, np, J, vc->dense, vc->linv, vc->d_status);
    const int64_t r0 = (int64_t)(J + 1) * PANEL, c0 = (int64_t)J * PANEL;
    const int m = (int)std::min(np - r0, band);
    if (m > 0) {
      double* Lp = vc->linvT + r0 * np + c0;
      BSR_TRY(dgemm128(true, m, PANEL, PANEL, 1.0, vc->dense + r0 * np + c0, np, vc->linv + c0 * np + c0, np, 0.0, Lp, np, 1, 0,
                       0, 0, 0, 0, st));
      BSR_TRY(dgemm128(true, m, m, PANEL, -1.0, Lp, np, Lp, np, 1.0, vc->dense + r0 * np + r0, np, 1, 0, 0, 0, 1, 0, st));
    }
  }
  // ---- X = L^-1: the diagonal 128-blocks are done; doubling: for the pair (X11, X22) of two consecutive inverted blocks
  // of size b, X21 = -X22 (L21 X11), with T = L21 X11 in the lower part of `dense`
  for (int64_t b = PANEL; b < np; b *= 2) {
    const int64_t step = 2 * b;
    const int nfull = (int)(np / step);                       // pairs with a full second block
    const int64_t rem = np - (int64_t)nfull * step;           // a last pair with a shorter second block, if rem > b
    auto pair = [&](int64_t r0, int64_t b2, int batch) -> int {
      const int64_t o21 = (r0 + b) * np + r0, o11 = r0 * np + r0, o22 = (r0 + b) * np + (r0 + b), sp = step * np + step;
      // L21 is banded: its row i is zero left of column b + i - band and entirely zero for i >= band, so T = L21 X11
      // has `mt` nonzero rows and the second product stops at k = mt
      const int64_t mt = std::min(b2, band);
      BSR_TRY(dgemm128(false, (int)mt, (int)b, (int)b, 1.0, vc->linvT + o21, np, vc->linv + o11, np, 0.0, vc->dense + o21, np,
                       batch, sp, sp, sp, 0, 1, st, (int)(b - band), 0));
      return dgemm128(false, (int)b2, (int)b, (int)b2, -1.0, vc->linv + o22, np, vc->dense + o21, np, 0.0, vc->linv + o21, np,
                      batch, sp, sp, sp, 0, 2, st, -(1 << 30), (int)mt);
    };
    if (nfull > 0) BSR_TRY(pair(0, b, nfull));
    if (rem > b) BSR_TRY(pair((int64_t)nfull * step, rem - b, 1));
  }
  LAUNCH(transpose_tile_kernel, dim3(nb, nb), tb, 0, st, np, vc->linv, vc->linvT);
  return BSR_OK;
}

static int coarse_solve(vcycle_t vc, const double* b, double* x, cudaStream_t st) {
  const unsigned grid = (unsigned)vc->nc;   // one CTA per row
  if (!grid) return BSR_OK;
  LAUNCH(trigemv_kernel, grid, TRIGEMV_THREADS, 0, st, vc->nc, vc->npad, vc->linv, b, vc->ytmp, 0);   // y = L^-1 b
  LAUNCH(trigemv_kernel, grid, TRIGEMV_THREADS, 0, st, vc->nc, vc->npad, vc->linvT, vc->ytmp, x, 1);  // x = L^-T y
  return BSR_OK;
}

// ------------------------------------------------------------------ the cycle
static int cycle(vcycle_t vc, int l, const double* b, double* x, cudaStream_t st) {
  if (l == vc->nlevels - 1) return coarse_solve(vc, b, x, st);
  Level& lv = vc->L[l];
  Level& nx = vc->L[l + 1];
  BSR_TRY(smooth(vc, l, b, x, true, st));                           // pre-smooth from the zero guess
  // r = b - A x as the plain SpMV plus one vector kernel: 0.340 + 0.012 ms on the 96^3 operator against 0.377 ms for the
  // SpMV with the subtraction in its epilogue (same rounding either way)
  BSR_TRY(spmv_launch(lv.A, x, lv.t, nullptr, EPI_ASSIGN, st));
  if (lv.n) LAUNCH(resid_kernel, (unsigned)((lv.n / 2 + 256) / 256), 256, 0, st, lv.n, b, lv.t, lv.r);
  BSR_TRY(transpose_ensure(lv.P, st));
  BSR_TRY(spmv_launch(lv.P->T, lv.r, nx.b, nullptr, EPI_ASSIGN, st)); // b_c = P^T r
  BSR_TRY(cycle(vc, l + 1, nx.b, nx.x, st));                         // coarse correction
  BSR_TRY(spmv_launch(lv.P, nx.x, x, nullptr, EPI_ADD, st));         // x += P x_c
  return smooth(vc, l, b, x, false, st);                             // post-smooth
}

// ------------------------------------------------------------------ PCG vector kernels (fixed-order reductions)
constexpr int DOT_BLOCKS = 592;  // 4 per SM on 148 SMs; fixed so that the summation order never changes

__global__ void __launch_bounds__(256)
dot_partial_kernel(int64_t n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ partial) {
  __shared__ double sh[8];
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    s = fma(a[i], b[i], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += sh[w];
    partial[blockIdx.x] = t;
  }
}

// out[0] = sum(partial) ; if hist != null also hist[0] = sqrt(sum)
__global__ void __launch_bounds__(32)
dot_final_kernel(int nparts, const double* __restrict__ partial, double* __restrict__ out, double* __restrict__ hist) {
  double s = 0.0;
  for (int i = threadIdx.x; i < nparts; i += 32) s += partial[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) {
    out[0] = s;
    if (hist) hist[0] = sqrt(s);
  }
}

// alpha = rz / pq ;  x += alpha p ;  r -= alpha q
__global__ void __launch_bounds__(256)
pcg_xr_kernel(int64_t n, const double* __restrict__ rz, const double* __restrict__ pq, const double* __restrict__ p,
              const double* __restrict__ q, double* __restrict__ x, double* __restrict__ r) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double alpha = rz[0] / pq[0];
  x[i] += alpha * p[i];
  r[i] -= alpha * q[i];
}

// beta = rz_new / rz ;  p = z + beta p
__global__ void __launch_bounds__(256)
pcg_p_kernel(int64_t n, const double* __restrict__ rz_new, const double* __restrict__ rz,
             const double* __restrict__ z, double* __restrict__ p) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double beta = rz_new[0] / rz[0];
  p[i] = z[i] + beta * p[i];
}

static int dot(vcycle_t vc, int64_t n, const double* a, const double* b, double* out, double* hist, cudaStream_t st) {
  LAUNCH(dot_partial_kernel, DOT_BLOCKS, 256, 0, st, n, a, b, vc->partial);
  LAUNCH(dot_final_kernel, 1, 32, 0, st, DOT_BLOCKS, vc->partial, out, hist);
  return BSR_OK;
}

static void vc_release(vcycle_t vc) {
  if (!vc) return;
  for (auto& lv : vc->L) { dev_free(lv.Dinv); dev_free(lv.r); dev_free(lv.t); dev_free(lv.d); dev_free(lv.b); dev_free(lv.x); }
  dev_free(vc->dense); dev_free(vc->linv); dev_free(vc->linvT); dev_free(vc->ytmp);
  dev_free(vc->coarse_rowidx); dev_free(vc->d_status); dev_free(vc->pr); dev_free(vc->pz); dev_free(vc->pp); dev_free(vc->pq);
  dev_free(vc->partial); dev_free(vc->scal);
  vc->magic = 0;
  delete vc;
}

static bool vc_ok(vcycle_t vc) { return vc && vc->magic == VC_MAGIC; }

}  // namespace bsramg

using namespace bsramg;


extern "C" {

int vcycle_refresh(vcycle_t vc, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemsetAsync(vc->d_status, 0, sizeof(int), st));
  for (int l = 0; l + 1 < vc->nlevels; ++l) {
    BSR_TRY(launch_dinv(vc->L[l], vc->d_status, st));
    BSR_TRY(transpose_ensure(vc->L[l].P, st));
  }
  NvtxRange nv("vcycle_refresh");
  return coarse_factor(vc, st);
}

int vcycle_status(vcycle_t vc, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  int h = 0;
  CUDA_TRY(cudaMemcpyAsync(&h, vc->d_status, sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  if (h & 1) return fail(BSR_ERR_NUMERIC, "singular or missing diagonal block");
  if (h & 2) return fail(BSR_ERR_NUMERIC, "coarsest operator is not positive definite");
  return BSR_OK;
}

int vcycle_create(vcycle_t* out, int32_t nlevels, const bsr_t* A, const bsr_t* P, const double* lambda_est,
                  int32_t cheb_degree, double lo, double hi, void* stream) {
  if (!out) return fail(BSR_ERR_NULL, "vcycle_create: out is null");
  *out = nullptr;
  if (nlevels < 1 || !A || (nlevels > 1 && (!P || !lambda_est))) return fail(BSR_ERR_NULL, "vcycle_create: null argument");
  if (cheb_degree < 1 || cheb_degree > 4 || !(hi > lo) || !(lo > 0)) return fail(BSR_ERR_SHAPE, "bad smoother parameters");
  for (int l = 0; l < nlevels; ++l) {
    if (!A[l] || A[l]->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle (A[%d])", l);
    if (A[l]->nbrows != A[l]->nbcols || A[l]->bs_r != A[l]->bs_c) return fail(BSR_ERR_SHAPE, "A[%d] is not square", l);
    if (l + 1 < nlevels) {
      if (!P[l] || P[l]->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle (P[%d])", l);
      if (P[l]->nbrows != A[l]->nbrows || P[l]->bs_r != A[l]->bs_r || P[l]->nbcols != A[l + 1]->nbrows ||
          P[l]->bs_c != A[l + 1]->bs_r)
        return fail(BSR_ERR_SHAPE, "P[%d] does not connect A[%d] and A[%d]", l, l, l + 1);
      if (!(lambda_est[l] > 0)) return fail(BSR_ERR_SHAPE, "lambda_est[%d] must be positive", l);
    }
  }
  bsr_t Ac = A[nlevels - 1];
  const int64_t nc = (int64_t)Ac->nbrows * Ac->bs_r;
  if (nc > 16384) return fail(BSR_ERR_LIMIT, "coarsest level has %lld unknowns (limit 16384)", (long long)nc);
  cudaStream_t st = (cudaStream_t)stream;
  vcycle_s* vc = new (std::nothrow) vcycle_s();
  if (!vc) return fail(BSR_ERR_ALLOC, "host allocation failed");
  vc->nlevels = nlevels; vc->degree = cheb_degree; vc->lo = lo; vc->hi = hi;
  vc->L.resize(nlevels);
  int rc = BSR_OK;
  for (int l = 0; l < nlevels && rc == BSR_OK; ++l) {
    Level& lv = vc->L[l];
    lv.A = A[l]; lv.P = (l + 1 < nlevels) ? P[l] : nullptr;
    lv.lambda = (l + 1 < nlevels) ? lambda_est[l] : 0.0;
    lv.bs = A[l]->bs_r;
    lv.n = (int64_t)A[l]->nbrows * lv.bs;
    if (l + 1 < nlevels) {
      rc = dev_alloc_t(&lv.Dinv, (size_t)lv.n * lv.bs);
      if (rc == BSR_OK) rc = dev_alloc_t(&lv.r, (size_t)lv.n);
      if (rc == BSR_OK) rc = dev_alloc_t(&lv.t, (size_t)lv.n);
      if (rc == BSR_OK) rc = dev_alloc_t(&lv.d, (size_t)lv.n);
    }
    if (l > 0 && rc == BSR_OK) {
      rc = dev_alloc_t(&lv.b, (size_t)lv.n);
      if (rc == BSR_OK) rc = dev_alloc_t(&lv.x, (size_t)lv.n);
    }
  }
  vc->nc = nc;
  vc->npad = ((nc + PANEL - 1) / PANEL) * PANEL;   // whole 128-wide panels (rows / columns >= nc carry the identity)
  if (vc->npad == 0) vc->npad = PANEL;
  const size_t np2 = (size_t)vc->npad * vc->npad;
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->dense, np2);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->linv, np2);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->linvT, np2);
  // the panel kernel's 180 KB of dynamic shared memory: opted in here, cold, on the device the hierarchy lives on
  if (rc == BSR_OK && cudaFuncSetAttribute(potrf_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PANEL_SMEM) != cudaSuccess)
    rc = fail(BSR_ERR_CUDA, "potrf_panel_kernel: cannot opt in to %d bytes of shared memory", PANEL_SMEM);
  if (rc == BSR_OK && cudaMemsetAsync(vc->linv, 0, np2 * 8, st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "memset failed");
  if (rc == BSR_OK && cudaMemsetAsync(vc->dense, 0, np2 * 8, st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "memset failed");
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->ytmp, (size_t)vc->npad);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->d_status, 1);
  const int64_t n0 = vc->L[0].n;
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->pr, (size_t)n0);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->pz, (size_t)n0);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->pp, (size_t)n0);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->pq, (size_t)n0);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->partial, (size_t)DOT_BLOCKS);
  if (rc == BSR_OK) rc = dev_alloc_t(&vc->scal, 8);
  if (rc == BSR_OK) {
    // block row of every stored block of the coarsest operator (for the dense fill)
    std::vector<int32_t> rowidx((size_t)Ac->nnzb);
    for (int32_t i = 0; i < Ac->nbrows; ++i)
      for (int32_t k = Ac->h_rowptr[i]; k < Ac->h_rowptr[(size_t)i + 1]; ++k) rowidx[(size_t)k] = i;
    rc = upload(&vc->coarse_rowidx, rowidx, st);
    // half-bandwidth of the coarsest operator in scalars, rounded up to whole panels
    int64_t hb = 0;
    for (int32_t i = 0; i < Ac->nbrows; ++i)
      for (int32_t k = Ac->h_rowptr[i]; k < Ac->h_rowptr[(size_t)i + 1]; ++k)
        hb = std::max<int64_t>(hb, std::abs((int64_t)Ac->h_colidx[(size_t)k] - i));
    vc->band = std::min<int64_t>(vc->npad, (((hb + 1) * Ac->bs_r + PANEL - 1) / PANEL) * PANEL);
    if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "upload failed");
  }
  if (rc == BSR_OK) {
    vc->magic = VC_MAGIC;
    rc = vcycle_refresh(vc, stream);
  }
  if (rc == BSR_OK) rc = vcycle_status(vc, stream);
  if (rc != BSR_OK) {
    vc_release(vc);
    return rc;
  }
  *out = vc;
  return BSR_OK;
}

int vcycle_apply(vcycle_t vc, const double* d_b, double* d_x, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  if (!d_b || !d_x) return fail(BSR_ERR_NULL, "null vector");
  NvtxRange nv("vcycle_apply");
  return cycle(vc, 0, d_b, d_x, (cudaStream_t)stream);
}

int vcycle_smooth(vcycle_t vc, int32_t level, const double* d_b, double* d_x, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  if (!d_b || !d_x) return fail(BSR_ERR_NULL, "null vector");
  if (level < 0 || level >= vc->nlevels - 1) return fail(BSR_ERR_SHAPE, "level %d has no smoother", level);
  return smooth(vc, level, d_b, d_x, false, (cudaStream_t)stream);
}

int pcg_solve(vcycle_t vc, const double* d_b, double* d_x, int32_t iters, double* d_resid_hist, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  if (!d_b || !d_x || !d_resid_hist) return fail(BSR_ERR_NULL, "null vector");
  if (iters < 0) return fail(BSR_ERR_SHAPE, "negative iteration count");
  cudaStream_t st = (cudaStream_t)stream;
  bsr_t A = vc->L[0].A;
  const int64_t n = vc->L[0].n;
  const unsigned grid = (unsigned)((n + 255) / 256);
  double *r = vc->pr, *z = vc->pz, *p = vc->pp, *q = vc->pq;
  double *rz = vc->scal + 0, *rz_new = vc->scal + 1, *pq = vc->scal + 2, *rr = vc->scal + 3;
  CUDA_TRY(cudaMemcpyAsync(r, d_b, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(cudaMemsetAsync(d_x, 0, (size_t)n * 8, st));
  BSR_TRY(dot(vc, n, r, r, rr, d_resid_hist, st));
  BSR_TRY(cycle(vc, 0, r, z, st));
  CUDA_TRY(cudaMemcpyAsync(p, z, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
  BSR_TRY(dot(vc, n, r, z, rz, nullptr, st));
  for (int k = 0; k < iters; ++k) {
    BSR_TRY(spmv_launch(A, p, q, nullptr, EPI_ASSIGN, st));
    BSR_TRY(dot(vc, n, p, q, pq, nullptr, st));
    if (grid) LAUNCH(pcg_xr_kernel, grid, 256, 0, st, n, rz, pq, p, q, d_x, r);
    BSR_TRY(dot(vc, n, r, r, rr, d_resid_hist + k + 1, st));
    BSR_TRY(cycle(vc, 0, r, z, st));
    BSR_TRY(dot(vc, n, r, z, rz_new, nullptr, st));
    if (grid) LAUNCH(pcg_p_kernel, grid, 256, 0, st, n, rz_new, rz, z, p);
    std::swap(rz, rz_new);
  }
  return BSR_OK;
}

int vcycle_apply_host(vcycle_t vc, const double* h_b, double* h_x, void* stream) {
  if (!vc_ok(vc)) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  if (!h_b || !h_x) return fail(BSR_ERR_NULL, "null vector");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)vc->L[0].n;
  // the PCG work vectors double as staging buffers
  CUDA_TRY(cudaMemcpyAsync(vc->pr, h_b, n * 8, cudaMemcpyHostToDevice, st));
  BSR_TRY(cycle(vc, 0, vc->pr, vc->pz, st));
  CUDA_TRY(cudaMemcpyAsync(h_x, vc->pz, n * 8, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return BSR_OK;
}

int vcycle_destroy(vcycle_t vc) {
  if (!vc) return BSR_OK;
  if (vc->magic != VC_MAGIC) return fail(BSR_ERR_NULL, "invalid vcycle handle");
  vc_release(vc);
  return BSR_OK;
}

}  // extern "C"
