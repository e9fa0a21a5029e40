// smooth.cu -- device prolongator smoothing P = (I - omega D^-1 A) P~ in blocks.
//
// "The tentative prolongator is improved by one step of a damped-Jacobi prolongator smoother,
// P = (I - omega D^-1 A) P~" (D the bs x bs block diagonal, reading R11).  PAPER.md:244: the cold setup is
// "dominated by symbolic coarsening and prolongator smoothing"; the smoother's MatAYPX with SUBSET_NONZERO_PATTERN
// "runs natively in blocks: the diagonal block is added directly ... adds block-for-block on device".
//
// Here the whole update is one pass over A: the pattern of P is the boolean pattern of A*P~ (cold, host,
// HostPlan::build_stage1 -- the same symbolic product ptap_symbolic uses for AP), the numeric phase is the staged
// <bf,bf,bc> product kernel of ptap_stream.cu with the update fused into its store:
//     P(i,J) = P~(i,J) [if stored] - omega * D_i^-1 * sum_j A(i,j) P~(j,J)
// so A*P~ is never written to memory and the block AXPY costs no extra pass.  D^-1 comes from the same block
// inversion kernel the V-cycle's point-block Jacobi uses.  A matrix outside the staged format runs a one-thread-per-
// output-block gather kernel with the same epilogue.  No atomics; fixed summation order.
#include <algorithm>

#include "internal.h"
#include "ptap_stream.h"

struct psmooth_plan_s {
  uint64_t magic = 0;
  bsr_t A = nullptr, Pt = nullptr;
  int64_t nnzb_a = 0, nnzb_pt = 0, nnzb_p = 0, nprod = 0;
  int32_t bf = 0, bc = 0, nbrows = 0, nbcols = 0;
  int32_t *rowptr_p = nullptr, *colidx_p = nullptr, *out_row = nullptr, *own_slot = nullptr;
  int32_t *pairptr = nullptr, *pstart = nullptr;   // gather fallback only
  void* pairs = nullptr;
  double* dinv = nullptr;
  int* status = nullptr;
  double *pw_v = nullptr, *pw_t = nullptr, *pw_part = nullptr, *pw_scal = nullptr;   // power iteration (first use)
  bsramg::StreamDev s1;
};
static const uint64_t PSM_MAGIC = 0x50534d4f4f544831ull;

namespace bsramg {

// gather fallback: one thread per output block, products in the plan's order, same epilogue as the staged kernel
template <int M, int N>
__global__ void __launch_bounds__(128)
smooth_gather_kernel(int32_t nout, const int32_t* __restrict__ out_row, const int32_t* __restrict__ own_slot,
                     const int32_t* __restrict__ rowptr_a, const int32_t* __restrict__ pstart,
                     const int32_t* __restrict__ pairptr, const uint32_t* __restrict__ pairs,
                     const double* __restrict__ avals, const double* __restrict__ tvals,
                     const double* __restrict__ dinv, double omega, double* __restrict__ pvals) {
  const int32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= nout) return;
  const int32_t row = __ldg(out_row + u);
  const int32_t x0 = __ldg(rowptr_a + row);
  double acc[M * N];
#pragma unroll
  for (int e = 0; e < M * N; ++e) acc[e] = 0.0;
  for (int32_t p = __ldg(pairptr + u); p < __ldg(pairptr + u + 1); ++p) {
    const uint32_t code = __ldg(pairs + p);
    const int32_t xs = x0 + (int32_t)(code & 0xffffu);
    const int32_t ys = __ldg(pstart + xs) + (int32_t)(code >> 16);
    const double* xb = avals + (int64_t)xs * M * M;
    const double* yb = tvals + (int64_t)ys * M * N;
#pragma unroll
    for (int r = 0; r < M; ++r)
#pragma unroll
      for (int m = 0; m < M; ++m) {
        const double xv = __ldg(xb + r * M + m);
#pragma unroll
        for (int c = 0; c < N; ++c) acc[r * N + c] = fma(xv, __ldg(yb + m * N + c), acc[r * N + c]);
      }
  }
  const double* di = dinv + (int64_t)row * M * M;
  const int32_t own = __ldg(own_slot + u);
  double* dst = pvals + (int64_t)u * M * N;
#pragma unroll
  for (int r = 0; r < M; ++r)
#pragma unroll
    for (int c = 0; c < N; ++c) {
      double t = 0.0;
#pragma unroll
      for (int m = 0; m < M; ++m) t = fma(__ldg(di + r * M + m), acc[m * N + c], t);
      dst[r * N + c] = fma(-omega, t, own >= 0 ? __ldg(tvals + (int64_t)own * M * N + r * N + c) : 0.0);
    }
}

template <int M, int N>
static int smooth_gather_launch(psmooth_plan_s* pl, double omega, double* d_vals_p, cudaStream_t st) {
  if (pl->nnzb_p == 0) return BSR_OK;
  const unsigned grid = (unsigned)((pl->nnzb_p + 127) / 128);
  LAUNCH((smooth_gather_kernel<M, N>), grid, 128, 0, st, (int32_t)pl->nnzb_p, pl->out_row, pl->own_slot,
         pl->A->d_rowptr, pl->pstart, pl->pairptr, (const uint32_t*)pl->pairs, pl->A->d_vals, pl->Pt->d_vals, pl->dinv,
         omega, d_vals_p);
  return BSR_OK;
}

// ---- lambda of D^-1 A by power iteration (reading R10), all on the device, fixed summation order
constexpr int PW_BLOCKS = 592;   // 4 per SM on 148 SMs; fixed so that the order of the norm's partial sums never changes

// w = D^-1 t in place (block row wise); partial[blockIdx] = sum of w^2 over this CTA's rows
template <int BS>
__global__ void __launch_bounds__(256)
dinv_apply_norm_kernel(int64_t nbrows, const double* __restrict__ dinv, double* __restrict__ t, double* __restrict__ partial) {
  __shared__ double sh[8];
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nbrows; i += (int64_t)gridDim.x * blockDim.x) {
    double r[BS], w[BS];
#pragma unroll
    for (int b = 0; b < BS; ++b) r[b] = t[i * BS + b];
#pragma unroll
    for (int a = 0; a < BS; ++a) {
      double z = 0.0;
#pragma unroll
      for (int b = 0; b < BS; ++b) z = fma(dinv[(i * BS + a) * BS + b], r[b], z);
      w[a] = z;
      s = fma(z, z, s);
    }
#pragma unroll
    for (int a = 0; a < BS; ++a) t[i * BS + a] = w[a];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tt = 0.0;
    for (int w = 0; w < 8; ++w) tt += sh[w];
    partial[blockIdx.x] = tt;
  }
}

__global__ void __launch_bounds__(256)
sumsq_partial_kernel(int64_t n, const double* __restrict__ v, double* __restrict__ partial) {
  __shared__ double sh[8];
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) s = fma(v[i], v[i], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tt = 0.0;
    for (int w = 0; w < 8; ++w) tt += sh[w];
    partial[blockIdx.x] = tt;
  }
}

// scal[0] = sqrt(sum(partial))
__global__ void __launch_bounds__(32)
norm_final_kernel(int nparts, const double* __restrict__ partial, double* __restrict__ scal) {
  double s = 0.0;
  for (int i = threadIdx.x; i < nparts; i += 32) s += partial[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) scal[0] = sqrt(s);
}

// v = w / scal[0]
__global__ void __launch_bounds__(256)
scale_by_norm_kernel(int64_t n, const double* __restrict__ w, const double* __restrict__ scal, double* __restrict__ v) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = w[i] / scal[0];
}

static void psmooth_release(psmooth_plan_s* pl) {
  if (!pl) return;
  dev_free(pl->pw_v); dev_free(pl->pw_t); dev_free(pl->pw_part); dev_free(pl->pw_scal);
  dev_free(pl->rowptr_p); dev_free(pl->colidx_p); dev_free(pl->out_row); dev_free(pl->own_slot);
  dev_free(pl->pairptr); dev_free(pl->pstart); dev_free(pl->pairs); dev_free(pl->dinv); dev_free(pl->status);
  stream_release(pl->s1);
  pl->magic = 0;
  delete pl;
}

static bool smooth_shape(int bf, int bc) {
  return (bf == 2 && bc == 3) || (bf == 3 && bc == 3) || (bf == 3 && bc == 6) || (bf == 6 && bc == 6);
}

}  // namespace bsramg

using namespace bsramg;

extern "C" {

int prolongator_smooth_symbolic(psmooth_plan_t* out, bsr_t A, bsr_t Pt, int64_t* nnzb_p, void* stream) {
  if (!out) return fail(BSR_ERR_NULL, "prolongator_smooth_symbolic: out is null");
  *out = nullptr;
  if (!A || !Pt || A->magic != BSR_MAGIC || Pt->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A->nbrows != A->nbcols || A->bs_r != A->bs_c) return fail(BSR_ERR_SHAPE, "A must be square with square blocks");
  if (A->nbcols != Pt->nbrows || A->bs_c != Pt->bs_r)
    return fail(BSR_ERR_SHAPE, "A (%d block cols, bs %d) does not match P~ (%d block rows, bs_r %d)", A->nbcols,
                A->bs_c, Pt->nbrows, Pt->bs_r);
  if (!smooth_shape(A->bs_r, Pt->bs_c)) return fail(BSR_ERR_BLOCK, "unsupported block shapes in prolongator smoothing");
  cudaStream_t st = (cudaStream_t)stream;
  HostPlan hp;
  int rc = hp.build_stage1(A->nbrows, A->h_rowptr.data(), A->h_colidx.data(), Pt->nbcols, Pt->h_rowptr.data(),
                           Pt->h_colidx.data());
  if (rc != BSR_OK) return fail(rc, "prolongator_smooth_symbolic: %s", hp.err.c_str());
  const int64_t np = (int64_t)hp.colidx_ap.size();
  if (np * A->bs_r * Pt->bs_c >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "P has 2^31 or more values");
  // own_slot: the tentative block with the same coordinate (the SUBSET pattern of the block AXPY)
  std::vector<int32_t> own((size_t)np, -1);
  int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
  for (int32_t i = 0; i < A->nbrows; ++i) {
    const int32_t* lo = hp.colidx_ap.data() + hp.rowptr_ap[i];
    const int32_t* hi = hp.colidx_ap.data() + hp.rowptr_ap[i + 1];
    for (int32_t q = Pt->h_rowptr[i]; q < Pt->h_rowptr[i + 1]; ++q) {
      const int32_t* it = std::lower_bound(lo, hi, Pt->h_colidx[q]);
      if (it == hi || *it != Pt->h_colidx[q]) bad |= 1;   // A has no diagonal block in row i
      else own[(size_t)(it - hp.colidx_ap.data())] = q;
    }
  }
  if (bad) return fail(BSR_ERR_STRUCTURE, "a block of P~ lies outside the pattern of A*P~ (A lacks a diagonal block)");
  psmooth_plan_s* pl = new (std::nothrow) psmooth_plan_s();
  if (!pl) return fail(BSR_ERR_ALLOC, "host allocation failed");
  pl->A = A; pl->Pt = Pt; pl->nnzb_a = A->nnzb; pl->nnzb_pt = Pt->nnzb; pl->nnzb_p = np;
  pl->nprod = (int64_t)hp.k1.size();
  pl->bf = A->bs_r; pl->bc = Pt->bs_c; pl->nbrows = A->nbrows; pl->nbcols = Pt->nbcols;
  rc = upload(&pl->rowptr_p, hp.rowptr_ap, st);
  if (rc == BSR_OK) rc = upload(&pl->colidx_p, hp.colidx_ap, st);
  if (rc == BSR_OK) rc = upload(&pl->out_row, hp.rowidx_ap, st);
  if (rc == BSR_OK) rc = upload(&pl->own_slot, own, st);
  if (rc == BSR_OK) rc = dev_alloc_t(&pl->dinv, (size_t)A->nbrows * A->bs_r * A->bs_r);
  if (rc == BSR_OK) rc = dev_alloc_t(&pl->status, 1);
  if (rc == BSR_OK && cudaMemsetAsync(pl->status, 0, sizeof(int), st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "memset failed");
  const Options opt = options();
  if (rc == BSR_OK && !opt.force_gather) {
    std::vector<StreamBrickDef> bricks;
    StreamPlan sp;
    const StreamShape sh{pl->bf, pl->bf, pl->bc};
    stream_bricks_stage1(hp, sh, opt.smem_stage1, A->h_rowptr.data(), A->h_colidx.data(), Pt->h_rowptr.data(), bricks);
    stream_build(sh, STREAM_THREADS_DIRECT / 32, opt.smem_stage1, bricks, A->h_rowptr.data(), A->h_colidx.data(),
                 Pt->h_rowptr.data(), hp.rowptr_ap.data(), hp.pairptr1.data(), hp.k1.data(), hp.q1.data(), sp);
    rc = stream_upload(sh, sp, pl->s1, st, /*smooth=*/true);
  }
  if (rc == BSR_OK && !pl->s1.ok) {
    std::vector<uint32_t> packed(hp.k1.size());
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < (int64_t)packed.size(); ++p) packed[(size_t)p] = hp.k1[(size_t)p] | ((uint32_t)hp.q1[(size_t)p] << 16);
    uint32_t* dp = nullptr;
    rc = upload(&pl->pairptr, hp.pairptr1, st);
    if (rc == BSR_OK) rc = upload(&pl->pstart, hp.pstart, st);
    if (rc == BSR_OK) rc = upload(&dp, packed, st);
    pl->pairs = dp;
    if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  }
  if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  if (rc != BSR_OK) { psmooth_release(pl); return rc; }
  pl->magic = PSM_MAGIC;
  if (nnzb_p) *nnzb_p = np;
  *out = pl;
  return BSR_OK;
}

int prolongator_smooth_structure(psmooth_plan_t pl, int32_t* d_rowptr_p, int32_t* d_colidx_p, void* stream) {
  if (!pl || pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!d_rowptr_p || (pl->nnzb_p && !d_colidx_p)) return fail(BSR_ERR_NULL, "null output array");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemcpyAsync(d_rowptr_p, pl->rowptr_p, ((size_t)pl->nbrows + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (pl->nnzb_p)
    CUDA_TRY(cudaMemcpyAsync(d_colidx_p, pl->colidx_p, (size_t)pl->nnzb_p * 4, cudaMemcpyDeviceToDevice, st));
  return BSR_OK;
}

int prolongator_smooth_numeric(psmooth_plan_t pl, bsr_t A, bsr_t Pt, double omega, double* d_vals_p, void* stream) {
  if (!pl || pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!A || !Pt || A->magic != BSR_MAGIC || Pt->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A != pl->A || Pt != pl->Pt || A->nnzb != pl->nnzb_a || Pt->nnzb != pl->nnzb_pt)
    return fail(BSR_ERR_PLAN, "plan was built from different matrices");
  if (!d_vals_p && pl->nnzb_p) return fail(BSR_ERR_NULL, "d_vals_p is null");
  if ((uintptr_t)d_vals_p & 15) return fail(BSR_ERR_ALIGN, "d_vals_p must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv("prolongator_smooth_numeric");
  BSR_TRY(block_diag_inverse(A, pl->dinv, pl->status, st));
  if (pl->s1.ok) {
    StreamArgs a = pl->s1.args;
    a.xvals = A->d_vals; a.yvals = Pt->d_vals; a.cvals = d_vals_p;
    a.dinv = pl->dinv; a.own_vals = Pt->d_vals; a.out_row = pl->out_row; a.own_slot = pl->own_slot; a.omega = omega;
    return stream_launch_smooth(pl->bf, pl->bc, a, pl->s1.nbricks, pl->s1.smem, st);
  }
  switch (pl->bf * 10 + pl->bc) {
    case 23: return smooth_gather_launch<2, 3>(pl, omega, d_vals_p, st);
    case 33: return smooth_gather_launch<3, 3>(pl, omega, d_vals_p, st);
    case 36: return smooth_gather_launch<3, 6>(pl, omega, d_vals_p, st);
    case 66: return smooth_gather_launch<6, 6>(pl, omega, d_vals_p, st);
  }
  return fail(BSR_ERR_BLOCK, "unsupported block shapes in prolongator smoothing");
}

int prolongator_smooth_lambda(psmooth_plan_t pl, bsr_t A, const double* d_v0, int32_t iters, double* lambda, void* stream) {
  if (!pl || pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!A || A->magic != BSR_MAGIC || A != pl->A) return fail(BSR_ERR_PLAN, "plan was built from a different matrix");
  if (!d_v0 || !lambda) return fail(BSR_ERR_NULL, "null argument");
  if (iters < 1) return fail(BSR_ERR_SHAPE, "iters must be positive");
  if ((uintptr_t)d_v0 & 15) return fail(BSR_ERR_ALIGN, "d_v0 must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv("prolongator_smooth_lambda");
  const int64_t n = (int64_t)A->nbrows * A->bs_r;
  if (!pl->pw_v) {   // cold: work vectors at first use
    BSR_TRY(dev_alloc_t(&pl->pw_v, (size_t)n));
    BSR_TRY(dev_alloc_t(&pl->pw_t, (size_t)n));
    BSR_TRY(dev_alloc_t(&pl->pw_part, (size_t)PW_BLOCKS));
    BSR_TRY(dev_alloc_t(&pl->pw_scal, 2));
  }
  BSR_TRY(block_diag_inverse(A, pl->dinv, pl->status, st));
  const unsigned gv = (unsigned)((n + 255) / 256);
  // v <- v0 / ||v0||
  LAUNCH(sumsq_partial_kernel, PW_BLOCKS, 256, 0, st, n, d_v0, pl->pw_part);
  LAUNCH(norm_final_kernel, 1, 32, 0, st, PW_BLOCKS, pl->pw_part, pl->pw_scal);
  LAUNCH(scale_by_norm_kernel, gv, 256, 0, st, n, d_v0, pl->pw_scal, pl->pw_v);
  for (int it = 0; it < iters; ++it) {
    BSR_TRY(spmv_launch(A, pl->pw_v, pl->pw_t, nullptr, EPI_ASSIGN, st));               // t = A v
    switch (A->bs_r) {                                                                  // w = D^-1 t, ||w||^2 partials
      case 2: LAUNCH(dinv_apply_norm_kernel<2>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, pl->dinv, pl->pw_t, pl->pw_part); break;
      case 3: LAUNCH(dinv_apply_norm_kernel<3>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, pl->dinv, pl->pw_t, pl->pw_part); break;
      case 6: LAUNCH(dinv_apply_norm_kernel<6>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, pl->dinv, pl->pw_t, pl->pw_part); break;
      default: return fail(BSR_ERR_BLOCK, "unsupported block size %d", A->bs_r);
    }
    LAUNCH(norm_final_kernel, 1, 32, 0, st, PW_BLOCKS, pl->pw_part, pl->pw_scal);        // lambda = ||w||
    LAUNCH(scale_by_norm_kernel, gv, 256, 0, st, n, pl->pw_t, pl->pw_scal, pl->pw_v);    // v = w / lambda
  }
  CUDA_TRY(cudaMemcpyAsync(lambda, pl->pw_scal, sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return BSR_OK;
}

int prolongator_smooth_status(psmooth_plan_t pl, void* stream) {
  if (!pl || pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  cudaStream_t st = (cudaStream_t)stream;
  int h = 0;
  CUDA_TRY(cudaMemcpyAsync(&h, pl->status, sizeof(int), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (h) return fail(BSR_ERR_NUMERIC, "singular or missing diagonal block in prolongator smoothing");
  return BSR_OK;
}

int prolongator_smooth_get_info(psmooth_plan_t pl, int64_t* n_products, int64_t* algorithmic_bytes, int32_t* staged) {
  if (!pl || pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (n_products) *n_products = pl->nprod;
  if (algorithmic_bytes) {
    auto bytes = [](int64_t nnzb, int br, int bc, int64_t nbrows) { return nnzb * (8LL * br * bc + 4) + 4LL * (nbrows + 1); };
    *algorithmic_bytes = bytes(pl->nnzb_a, pl->bf, pl->bf, pl->nbrows) + bytes(pl->nnzb_pt, pl->bf, pl->bc, pl->nbrows) +
                         bytes(pl->nnzb_p, pl->bf, pl->bc, pl->nbrows);
  }
  if (staged) *staged = pl->s1.ok ? 1 : 0;
  return BSR_OK;
}

int prolongator_smooth_destroy(psmooth_plan_t pl) {
  if (!pl) return BSR_OK;
  if (pl->magic != PSM_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  psmooth_release(pl);
  return BSR_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ the power iteration without any allocation
// bsr_lambda_noalloc: prolongator_smooth_lambda's iteration (same kernels, same order, same bits) for callers that may
// not allocate -- code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  Its work space
// (D^-1, the two work vectors, the norm's partial sums, the status word) is a fixed file-scope device array: every GPU
// that loads the library holds BSR_NOALLOC_SCRATCH_BYTES (32 MiB) until exit.  In HOST code the array's name is only a
// handle for the runtime, not a device address: the pointer the kernels get comes from cudaGetSymbolAddress, looked up
// once per device with that device current.
namespace bsramg {

constexpr int64_t NOALLOC_DOUBLES = BSR_NOALLOC_SCRATCH_BYTES / 8;
static __device__ __align__(256) double noalloc_scratch[NOALLOC_DOUBLES];

constexpr int NOALLOC_MAX_DEVICES = 64;
static std::atomic<double*> noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of the array, per device ordinal

static int noalloc_base(double** out) {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(BSR_ERR_LIMIT, "device ordinal %d outside the table", dev);
  double* p = noalloc_ptr[dev].load(std::memory_order_acquire);
  if (!p) {   // set-up, once per device (idempotent: two racing threads obtain the same address)
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), noalloc_scratch);
    if (e != cudaSuccess || !p) return fail(BSR_ERR_CUDA, "cudaGetSymbolAddress(noalloc_scratch): %s", cudaGetErrorString(e));
    noalloc_ptr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return BSR_OK;
}

static int64_t up32(int64_t doubles) { return (doubles + 31) & ~int64_t(31); }   // segments start on 256 bytes

}  // namespace bsramg

extern "C" int bsr_lambda_noalloc_scratch_doubles(int32_t nbrows, int32_t bs, int64_t* doubles) {
  if (!doubles) return fail(BSR_ERR_NULL, "null output");
  if (nbrows < 0 || bs < 1) return fail(BSR_ERR_SHAPE, "bad size");
  const int64_t n = (int64_t)nbrows * bs;
  *doubles = up32(n * bs) + 2 * up32(n) + up32(PW_BLOCKS) + 32 /* lambda */ + 32 /* status */;
  return BSR_OK;
}

extern "C" int bsr_lambda_noalloc(bsr_t A, const double* d_v0, int32_t iters, double* d_lambda, int32_t* d_status,
                                  void* stream) {
  if (!A || A->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (!d_v0 || !d_lambda) return fail(BSR_ERR_NULL, "null argument");
  if (A->nbrows != A->nbcols || A->bs_r != A->bs_c) return fail(BSR_ERR_SHAPE, "A must be square with square blocks");
  if (A->bs_r != 2 && A->bs_r != 3 && A->bs_r != 6) return fail(BSR_ERR_BLOCK, "unsupported block size %d", A->bs_r);
  if (iters < 1) return fail(BSR_ERR_SHAPE, "iters must be positive");
  if ((uintptr_t)d_v0 & 15) return fail(BSR_ERR_ALIGN, "d_v0 must be 16-byte aligned");
  int64_t need = 0;
  BSR_TRY(bsr_lambda_noalloc_scratch_doubles(A->nbrows, A->bs_r, &need));
  if (need > NOALLOC_DOUBLES)
    return fail(BSR_ERR_LIMIT, "bsr_lambda_noalloc: %d block rows of size %d need %lld bytes of work space, the fixed array "
                "holds %lld (BSR_NOALLOC_SCRATCH_BYTES); use prolongator_smooth_lambda", A->nbrows, A->bs_r,
                (long long)(need * 8), (long long)BSR_NOALLOC_SCRATCH_BYTES);
  if (A->nbrows == 0) return fail(BSR_ERR_SHAPE, "empty matrix");
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv("bsr_lambda_noalloc");
  double* base = nullptr;
  BSR_TRY(noalloc_base(&base));
  const int64_t n = (int64_t)A->nbrows * A->bs_r;
  double* dinv = base;
  double* v = dinv + up32(n * A->bs_r);
  double* t = v + up32(n);
  double* part = t + up32(n);
  double* scal = part + up32(PW_BLOCKS);
  int* status = reinterpret_cast<int*>(scal + 32);
  // the array keeps the last call's contents: the status word is OR-ed into, so it must start at zero; D^-1, v, t and
  // the partial sums are written in full before they are read
  CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int), st));
  BSR_TRY(block_diag_inverse(A, dinv, status, st));
  const unsigned gv = (unsigned)((n + 255) / 256);
  LAUNCH(sumsq_partial_kernel, PW_BLOCKS, 256, 0, st, n, d_v0, part);
  LAUNCH(norm_final_kernel, 1, 32, 0, st, PW_BLOCKS, part, scal);
  LAUNCH(scale_by_norm_kernel, gv, 256, 0, st, n, d_v0, scal, v);                         // v <- v0 / ||v0||
  for (int it = 0; it < iters; ++it) {
    BSR_TRY(spmv_launch(A, v, t, nullptr, EPI_ASSIGN, st));                                // t = A v
    switch (A->bs_r) {                                                                    // w = D^-1 t, ||w||^2 partials
      case 2: LAUNCH(dinv_apply_norm_kernel<2>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, dinv, t, part); break;
      case 3: LAUNCH(dinv_apply_norm_kernel<3>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, dinv, t, part); break;
      default: LAUNCH(dinv_apply_norm_kernel<6>, PW_BLOCKS, 256, 0, st, (int64_t)A->nbrows, dinv, t, part); break;
    }
    LAUNCH(norm_final_kernel, 1, 32, 0, st, PW_BLOCKS, part, scal);                        // lambda = ||w||
    LAUNCH(scale_by_norm_kernel, gv, 256, 0, st, n, t, scal, v);                           // v = w / lambda
  }
  CUDA_TRY(cudaMemcpyAsync(d_lambda, scal, sizeof(double), cudaMemcpyDeviceToDevice, st));
  if (d_status) CUDA_TRY(cudaMemcpyAsync(d_status, status, sizeof(int), cudaMemcpyDeviceToDevice, st));
  return BSR_OK;
}
