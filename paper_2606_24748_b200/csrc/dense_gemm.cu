// dense_gemm.cu -- fp64 tensor-core (DMMA) GEMM for the coarsest-level factorisation (vcycle_refresh).
//
// The coarsest operator of the V-cycle is "solved dense on device" (BASELINE.json config 4; reading R17):
// a blocked Cholesky factorisation and the explicit triangular inverse that turns every later solve into two
// mat-vecs.  Both are built from ONE kernel, C = beta*C + alpha * A * op(B) on 128x128 tiles: 256 threads, k in chunks of
// 16 through shared memory with the next chunk prefetched into registers, and the products on the fp64 tensor-core path
// (mma.sync m8n8k4, DMMA): a warp owns a 32x64 piece of the tile as 4x8 fragments of 8x8, so a k-step of 4 costs 12
// 8-byte shared-memory loads per lane for 32 MMAs.  The DMMA rate equals the plain FMA rate on this part (37 TFLOP/s
// either way, measured); what the tensor path buys is operand traffic: the register-tiled FMA version of this kernel
// (8x8 per thread) needed 8 LDS.128 per 64 FMAs, which kept the shared-memory pipe as busy as the fp64 pipe and held
// the kernel to ~12.5 TFLOP/s.  Triangular and banded operands arrive as k-ranges per tile.
// All matrices are row-major; m and n multiples of 128, k ranges multiples of 16 (the caller pads).
#include "internal.h"

namespace bsramg {

constexpr int GK = 16;   // k-chunk

// GT: the CTA's tile (128; 64 or 32 for launches that would leave most SMs without a larger tile); 2 GT threads
template <int GT, bool TRANSB>
__global__ void __launch_bounds__(2 * GT)
dgemm128_kernel(int k, double alpha, const double* __restrict__ A, int64_t lda, const double* __restrict__ B,
                int64_t ldb, double beta, double* __restrict__ C, int64_t ldc, int64_t sA, int64_t sB, int64_t sC,
                int tri, int klim, int koff, int kcap) {
  const int m0 = blockIdx.y * GT, n0 = blockIdx.x * GT;
  if (tri && n0 > m0) return;                       // lower tiles only
  A += (int64_t)blockIdx.z * sA; B += (int64_t)blockIdx.z * sB; C += (int64_t)blockIdx.z * sC;
  int kbeg = 0, kend = k;
  if (klim == 1) kbeg = min(n0, k);                 // B (k x n) is lower triangular: rows k < n0 of this tile are zero
  if (klim == 2) kend = min(m0 + GT, k);            // A (m x k) is lower triangular: columns k >= m0+128 are zero
  kbeg = max(kbeg, min((koff + m0) & ~(GK - 1), k));   // A banded: row m0 + i is zero left of column koff + m0 + i
  kend = min(kend, kcap);                           // B has no nonzero row at or beyond kcap
  constexpr int GS = GT + 4;                        // padded shared-memory row: fragment loads hit 16 distinct banks
  constexpr int NJ = GT / 16;                       // 8x8 fragments across the warp's piece (32 x GT/2)
  __shared__ __align__(16) double As[GK][GS];
  __shared__ __align__(16) double Bs[GK][GS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = (warp % (GT / 32)) * 32, wn = (warp / (GT / 32)) * (GT / 2);   // this warp's 32 x GT/2 piece
  const int fk = lane & 3, fr = lane >> 2;                     // fragment coordinates of this lane
  double acc[4][NJ][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  // staging roles: A (and B when TRANSB): row tid/2, eight k values at (tid&1)*8;  B (k x n): k rows bk and bk + 8,
  // four columns each
  const int ar = tid >> 1, ak = (tid & 1) * 8;
  const int bk = tid / (GT / 4), bc = (tid % (GT / 4)) * 4;
  const double* ap = A + (int64_t)(m0 + ar) * lda + ak;
  const double* bp = TRANSB ? B + (int64_t)(n0 + ar) * ldb + ak : B + (int64_t)bk * ldb + n0 + bc;
  double2 pa[4], pb[4];
  auto fetch = [&](int kk) {
#pragma unroll
    for (int u = 0; u < 4; ++u) pa[u] = *reinterpret_cast<const double2*>(ap + kk + 2 * u);
    if (TRANSB) {
#pragma unroll
      for (int u = 0; u < 4; ++u) pb[u] = *reinterpret_cast<const double2*>(bp + kk + 2 * u);
    } else {
      pb[0] = *reinterpret_cast<const double2*>(bp + (int64_t)kk * ldb);
      pb[1] = *reinterpret_cast<const double2*>(bp + (int64_t)kk * ldb + 2);
      pb[2] = *reinterpret_cast<const double2*>(bp + (int64_t)(kk + 8) * ldb);
      pb[3] = *reinterpret_cast<const double2*>(bp + (int64_t)(kk + 8) * ldb + 2);
    }
  };
  if (kbeg < kend) fetch(kbeg);
  for (int kk = kbeg; kk < kend; kk += GK) {
#pragma unroll
    for (int u = 0; u < 4; ++u) { As[ak + 2 * u][ar] = pa[u].x; As[ak + 2 * u + 1][ar] = pa[u].y; }
    if (TRANSB) {
#pragma unroll
      for (int u = 0; u < 4; ++u) { Bs[ak + 2 * u][ar] = pb[u].x; Bs[ak + 2 * u + 1][ar] = pb[u].y; }
    } else {
      *reinterpret_cast<double2*>(&Bs[bk][bc]) = pb[0];
      *reinterpret_cast<double2*>(&Bs[bk][bc + 2]) = pb[1];
      *reinterpret_cast<double2*>(&Bs[bk + 8][bc]) = pb[2];
      *reinterpret_cast<double2*>(&Bs[bk + 8][bc + 2]) = pb[3];
    }
    __syncthreads();
    if (kk + GK < kend) fetch(kk + GK);             // next chunk in flight while this one is multiplied
#pragma unroll
    for (int q = 0; q < GK; q += 4) {
      double af[4], bf[NJ];
#pragma unroll
      for (int i = 0; i < 4; ++i) af[i] = As[q + fk][wm + 8 * i + fr];
#pragma unroll
      for (int j = 0; j < NJ; ++j) bf[j] = Bs[q + fk][wn + 8 * j + fr];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < NJ; ++j)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                       : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(af[i]), "d"(bf[j]));
    }
    __syncthreads();
  }
  // fragment (i, j): row 8 i + lane / 4, columns 8 j + 2 (lane % 4) + {0, 1}
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    double* crow = C + (int64_t)(m0 + wm + 8 * i + fr) * ldc + n0 + wn + 2 * fk;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      double2* cp = reinterpret_cast<double2*>(crow + 8 * j);
      double2 v = make_double2(alpha * acc[i][j][0], alpha * acc[i][j][1]);
      if (beta != 0.0) {
        const double2 o = *cp;
        v.x = fma(beta, o.x, v.x);
        v.y = fma(beta, o.y, v.y);
      }
      *cp = v;
    }
  }
}

int dgemm128(bool transB, int m, int n, int k, double alpha, const double* A, int64_t lda, const double* B, int64_t ldb,
             double beta, double* C, int64_t ldc, int batch, int64_t sA, int64_t sB, int64_t sC, int tri, int klim,
             cudaStream_t st, int koff, int kcap) {
  if (m <= 0 || n <= 0 || batch <= 0) return BSR_OK;
  if (m % 128 || n % 128 || k % GK || (lda & 1) || (ldb & 1) || (ldc & 1))
    return fail(BSR_ERR_SHAPE, "dgemm128: sizes must be multiples of the tile (m %d n %d k %d)", m, n, k);
  if (kcap <= 0 || kcap > k) kcap = k;
  if (koff < -(1 << 29)) koff = -(1 << 29);
  // a tile runs on ONE SM (64 fp64 FMAs per clock: a 64x64x128 tile is 4 us of arithmetic alone) and a grid runs in
  // waves of 148 tiles: take the largest tile that still gives four waves (measured at 6000 unknowns: 128-tiles from one
  // wave on 4.53 ms per refresh, from four waves on 4.35, the same rule for the 64-tiles 4.31)
  auto tiles = [&](int gt) { return (int64_t)(m / gt) * (tri ? (n / gt + 1) / 2 : n / gt) * batch; };
  const int gt = tiles(128) >= 592 ? 128 : tiles(64) >= 592 ? 64 : 32;
  const dim3 grid((unsigned)(n / gt), (unsigned)(m / gt), (unsigned)batch);
#define DGEMM_LAUNCH(GT, TB) \
  LAUNCH((dgemm128_kernel<GT, TB>), grid, 2 * GT, 0, st, k, alpha, A, lda, B, ldb, beta, C, ldc, sA, sB, sC, tri, klim, koff, kcap)
  if (gt == 32)      { if (transB) DGEMM_LAUNCH(32, true); else DGEMM_LAUNCH(32, false); }
  else if (gt == 64) { if (transB) DGEMM_LAUNCH(64, true); else DGEMM_LAUNCH(64, false); }
  else               { if (transB) DGEMM_LAUNCH(128, true); else DGEMM_LAUNCH(128, false); }
#undef DGEMM_LAUNCH
  return BSR_OK;
}

}  // namespace bsramg
