// assembly.cu -- blocked COO assembly of a BSR matrix and its finite-element driver.
//
// "the caller supplies, once, the (i,j) coordinates of every contribution ... builds a cached ...
// scatter plan, and thereafter each numeric assembly is a single MatSetValuesCOO that scatters a flat value array and
// sums duplicates, entirely on the device.  We generalize this to blocks ... each coordinate addresses a dense
// bs_r x bs_c block ... The block size need not be square".  PAPER.md:248-250: "the value stream is a sequence of
// dense blocks (square or rectangular), and the scatter writes and sums contiguous bs_r*bs_c runs"; finite-element
// assembly, "where per-element dense matrices generate exactly such a stream of duplicated ... contributions", is
// named as the next application.
//
// bcoo_plan_create (COLD) builds the sorted-unique map once: the matrix structure (one block per distinct coordinate,
// columns strictly ascending) and, per destination block, the ordered list of stream positions that carry its
// coordinate -- the duplicate-summation map in GATHER form.  bcoo_set_values (HOT) is one kernel: every destination
// value is the sum of its contributions in declaration order, read as contiguous bs_r*bs_c runs of the stream and
// written once.  No atomics, bit-reproducible.  The fem_q1_* calls are the driver for Q1 elasticity: 4^d block
// contributions per element, scaled by the element's modulus on the device.
#include <algorithm>
#include <numeric>

#include "internal.h"

struct bcoo_plan_s {
  uint64_t magic = 0;
  int64_t n = 0, nnzb = 0;
  int32_t nbrows = 0, nbcols = 0, bs_r = 0, bs_c = 0;
  int32_t *rowptr = nullptr, *colidx = nullptr, *segptr = nullptr, *perm = nullptr;
  int32_t* ctas = nullptr;   // staged kernel: per run {first block, blocks, first contribution, contributions}
  int64_t nctas = 0;         // runs; 0: a block with more contributions than a buffer holds -> the per-value kernel
};
static const uint64_t BCOO_MAGIC = 0x42434f4f504c414eull;

namespace bsramg {

// one thread per destination value: consecutive threads read consecutive doubles of the same contribution block
template <int BB>
__global__ void __launch_bounds__(256)
bcoo_sum_kernel(int64_t nvals, const int32_t* __restrict__ segptr, const int32_t* __restrict__ perm,
                const double* __restrict__ stream, double* __restrict__ vals) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nvals) return;
  const int64_t slot = t / BB;
  const int e = (int)(t - slot * BB);
  const int32_t p0 = __ldg(segptr + slot), p1 = __ldg(segptr + slot + 1);
  double s = 0.0;
  // up to four contributions in flight (positions first, then values; indices clamped instead of predicated so that
  // the loads are issued back to back), added in declaration order
  for (int32_t p = p0; p < p1; p += 4) {
    int32_t q[4];
    double v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) q[u] = __ldg(perm + min(p + u, p1 - 1));
#pragma unroll
    for (int u = 0; u < 4; ++u) v[u] = __ldg(stream + (int64_t)q[u] * BB + e);
#pragma unroll
    for (int u = 0; u < 4; ++u) s += (p + u < p1) ? v[u] : 0.0;
  }
  vals[t] = s;
}

// The same sums, a CTA at a time.  The per-value kernel above walks segment pointer -> stream position -> value once
// per thread, and of the three dependent latencies only the last moves bytes.  Here the plan cuts the destination
// blocks into runs whose contributions fill a CTA's shared memory (BCOO_ITEMS doubles, at most BCOO_NBMAX blocks); the
// CTA fetches the run's segment pointers and stream positions with two coalesced loads, every thread then has up to 16
// independent value loads to issue (two rounds of 8), parked in shared memory in contribution order, and one thread
// per destination value adds its segment in declaration order (the order of the kernel above and of the oracle:
// bit-identical) and stores coalesced.  4.47 -> 4.04 ms at config 3 (0.55 of the HBM peak).  A persistent variant
// (two 32 KB buffers per CTA, values by LDGSTS, the next run's indices fetched in their shadow) measured 4.33 ms and
// was not kept: the index latencies are not what binds this gather -- its reads are 72-byte pieces of the element
// stream, every 4.6 KB element record visited at four different times.
constexpr int BCOO_ITEMS = 8192;    // doubles of contributions a CTA parks (64 KB: three CTAs per SM)
constexpr int BCOO_NBMAX = 512;     // destination blocks per run
constexpr int BCOO_THREADS = 512;
constexpr size_t BCOO_FLAT_SMEM = (size_t)BCOO_ITEMS * 8 + (size_t)(BCOO_NBMAX + 4) * 4 + (size_t)(BCOO_ITEMS / 4) * 4;

template <int BB>
__global__ void __launch_bounds__(BCOO_THREADS)
bcoo_flat_kernel(const int4* __restrict__ runs, const int32_t* __restrict__ segptr, const int32_t* __restrict__ perm,
                 const double* __restrict__ stream, double* __restrict__ vals) {
  extern __shared__ __align__(16) unsigned char bcoo_smem[];
  double* part = reinterpret_cast<double*>(bcoo_smem);
  int32_t* seg = reinterpret_cast<int32_t*>(bcoo_smem + (size_t)BCOO_ITEMS * 8);
  int32_t* pos = seg + BCOO_NBMAX + 4;
  const int tid = threadIdx.x;
  const int4 c = __ldg(runs + blockIdx.x);                   // {first block, blocks, first contribution, contributions}
  const int b0 = c.x, nb = c.y, k0 = c.z, nk = c.w;
  for (int i = tid; i <= nb; i += BCOO_THREADS) seg[i] = __ldg(segptr + b0 + i) - k0;
  for (int i = tid; i < nk; i += BCOO_THREADS) pos[i] = __ldg(perm + k0 + i);
  __syncthreads();
  const int items = nk * BB;
  for (int base = tid; base < items; base += BCOO_THREADS * 8) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int it = base + u * BCOO_THREADS;
      const int k = it / BB, e = it - k * BB;
      v[u] = 0.0;
      if (it < items) v[u] = __ldg(stream + (int64_t)pos[k] * BB + e);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int it = base + u * BCOO_THREADS;
      if (it < items) part[it] = v[u];
    }
  }
  __syncthreads();
  for (int o = tid; o < nb * BB; o += BCOO_THREADS) {
    const int bl = o / BB, e = o - bl * BB;
    double s = 0.0;
    for (int k = seg[bl]; k < seg[bl + 1]; ++k) s += part[k * BB + e];
    vals[(int64_t)b0 * BB + o] = s;
  }
}

// dst block t = src block idx[t] (bs doubles each): packs halo entries / prolongator rows for an exchange
__global__ void __launch_bounds__(256)
gather_blocks_kernel(int64_t nvals, int bs, const int32_t* __restrict__ idx, const double* __restrict__ src,
                     double* __restrict__ dst) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nvals) return;
  const int64_t b = t / bs;
  dst[t] = __ldg(src + (int64_t)__ldg(idx + b) * bs + (t - b * bs));
}

// dst block idx[t] += src block t (idx holds distinct blocks: no two threads touch the same value, no atomics)
__global__ void __launch_bounds__(256)
scatter_add_blocks_kernel(int64_t nvals, int bs, const int32_t* __restrict__ idx, const double* __restrict__ src,
                          double* __restrict__ dst) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nvals) return;
  const int64_t b = t / bs;
  dst[(int64_t)__ldg(idx + b) * bs + (t - b * bs)] += __ldg(src + t);
}

// ---- Q1 elasticity driver: element e = ex + ne*(ey + ne*ez), local node a has offset bit k of a in direction k
__device__ __forceinline__ void q1_nodes(int d, int ne, int64_t e, int a, int b, int& ia, int& ib, int (&ca)[3], int (&cb)[3]) {
  const int n = ne + 1;
  const int ex = (int)(e % ne), ey = (int)((e / ne) % ne), ez = (d == 3) ? (int)(e / ((int64_t)ne * ne)) : 0;
  ca[0] = ex + (a & 1); ca[1] = ey + ((a >> 1) & 1); ca[2] = ez + ((a >> 2) & 1);
  cb[0] = ex + (b & 1); cb[1] = ey + ((b >> 1) & 1); cb[2] = ez + ((b >> 2) & 1);
  ia = ca[0] + n * (ca[1] + n * ca[2]);
  ib = cb[0] + n * (cb[1] + n * cb[2]);
}

__global__ void __launch_bounds__(256)
q1_coords_kernel(int d, int ne, int64_t e0, int64_t ncontrib, int32_t* __restrict__ brow, int32_t* __restrict__ bcol) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncontrib) return;
  const int nen = 1 << d, nn = nen * nen;
  const int64_t e = e0 + c / nn;
  const int ab = (int)(c % nn), a = ab / nen, b = ab % nen;
  int ia, ib, ca[3], cb[3];
  q1_nodes(d, ne, e, a, b, ia, ib, ca, cb);
  brow[c] = ia;
  bcol[c] = ib;
}

// stream block c = E_e * Ke[a][b] (d x d); with `dirichlet` the face ix = 0 is clamped in the stream itself
// (reading R4): a block whose row or column node is clamped is zero, except the node's own diagonal block,
// which carries I / (number of elements adjacent to the node) so that the assembled block is exactly I.
// One thread per contribution block: the element / local-node arithmetic is done once per block, the reference element
// matrix sits in shared memory; the CTA's 256 blocks go through shared memory so that the stream is written with
// fully coalesced stores.
template <int D>
__global__ void __launch_bounds__(256)
q1_blocks_kernel(int ne, int64_t e0, int64_t ncontrib, const double* __restrict__ Ke, const double* __restrict__ E,
                 int dirichlet, double* __restrict__ stream) {
  constexpr int NEN = 1 << D, NN = NEN * NEN, BB = D * D, ND = D * NEN;
  __shared__ double ke[ND * ND];
  __shared__ double outb[256 * BB];
  for (int t = threadIdx.x; t < ND * ND; t += blockDim.x) ke[t] = Ke[t];
  __syncthreads();
  const int64_t c0 = (int64_t)blockIdx.x * blockDim.x;
  const int64_t c = c0 + threadIdx.x;
  const bool live = c < ncontrib;
  if (live) {
  const int64_t e = e0 + c / NN;
  const int ab = (int)(c % NN), a = ab / NEN, b = ab % NEN;
  const double Ee = E ? __ldg(E + e) : 1.0;
  double v[BB];
#pragma unroll
  for (int i = 0; i < D; ++i)
#pragma unroll
    for (int j = 0; j < D; ++j) v[i * D + j] = Ee * ke[(a * D + i) * ND + (b * D + j)];
  if (dirichlet) {
    int ia, ib, ca[3], cb[3];
    q1_nodes(D, ne, e, a, b, ia, ib, ca, cb);
    if (ca[0] == 0 || cb[0] == 0) {
#pragma unroll
      for (int t = 0; t < BB; ++t) v[t] = 0.0;
      if (a == b) {
        const int cy = (ca[1] > 0 && ca[1] < ne) ? 2 : 1;
        const int cz = (D == 3 && ca[2] > 0 && ca[2] < ne) ? 2 : 1;
#pragma unroll
        for (int i = 0; i < D; ++i) v[i * D + i] = 1.0 / (double)(cy * cz);
      }
    }
  }
#pragma unroll
  for (int t = 0; t < BB; ++t) outb[threadIdx.x * BB + t] = v[t];   // odd stride (9) / 4: conflict-free enough
  }
  __syncthreads();
  const int64_t nlive = min((int64_t)blockDim.x, ncontrib - c0) * BB;
  double* dst = stream + c0 * BB;
  for (int64_t t = threadIdx.x; t < nlive; t += blockDim.x) dst[t] = outb[t];
}

static void bcoo_release(bcoo_plan_s* pl) {
  if (!pl) return;
  dev_free(pl->rowptr); dev_free(pl->colidx); dev_free(pl->segptr); dev_free(pl->perm); dev_free(pl->ctas);
  pl->magic = 0;
  delete pl;
}

}  // namespace bsramg

using namespace bsramg;

extern "C" {

int bcoo_plan_create(bcoo_plan_t* out, int64_t n, const int32_t* d_brow, const int32_t* d_bcol, int32_t nbrows,
                     int32_t nbcols, int32_t bs_r, int32_t bs_c, int64_t* nnzb_out, void* stream) {
  if (!out) return fail(BSR_ERR_NULL, "bcoo_plan_create: out is null");
  *out = nullptr;
  if (n < 0 || nbrows < 0 || nbcols < 0) return fail(BSR_ERR_SHAPE, "negative size");
  if (n > 0 && (!d_brow || !d_bcol)) return fail(BSR_ERR_NULL, "null coordinate array");
  if (!shape_supported(bs_r, bs_c)) return fail(BSR_ERR_BLOCK, "unsupported block shape %dx%d", bs_r, bs_c);
  if (n >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "2^31 or more contributions");
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<int32_t> br((size_t)n), bc((size_t)n);
  if (n) {
    CUDA_TRY(cudaMemcpyAsync(br.data(), d_brow, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(bc.data(), d_bcol, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
  }
  // counting sort of the contributions by block row (stable: declaration order inside a row)
  std::vector<int64_t> rstart((size_t)nbrows + 1, 0);
  int bad = 0;
  int64_t nkept = 0;   // a contribution with a negative coordinate is declared but ignored (the COO convention)
  for (int64_t c = 0; c < n; ++c) {
    if (br[(size_t)c] < 0 || bc[(size_t)c] < 0) continue;
    if (br[(size_t)c] >= nbrows || bc[(size_t)c] >= nbcols) { bad = 1; break; }
    rstart[(size_t)br[(size_t)c] + 1]++;
    ++nkept;
  }
  if (bad) return fail(BSR_ERR_STRUCTURE, "block coordinate out of range");
  for (int32_t i = 0; i < nbrows; ++i) rstart[(size_t)i + 1] += rstart[(size_t)i];
  std::vector<int32_t> byrow((size_t)nkept);
  {
    std::vector<int64_t> fill(rstart.begin(), rstart.end() - 1);
    for (int64_t c = 0; c < n; ++c)
      if (br[(size_t)c] >= 0 && bc[(size_t)c] >= 0) byrow[(size_t)fill[(size_t)br[(size_t)c]]++] = (int32_t)c;
  }
  // inside each row: order by (column, declaration index); distinct columns become the row's blocks
  std::vector<int32_t> nblk((size_t)nbrows, 0);
#pragma omp parallel for schedule(dynamic, 1024)
  for (int32_t i = 0; i < nbrows; ++i) {
    int32_t* lo = byrow.data() + rstart[(size_t)i];
    int32_t* hi = byrow.data() + rstart[(size_t)i + 1];
    std::sort(lo, hi, [&](int32_t u, int32_t v) { return bc[(size_t)u] != bc[(size_t)v] ? bc[(size_t)u] < bc[(size_t)v] : u < v; });
    int32_t cnt = 0;
    for (int32_t* p = lo; p < hi; ++p)
      if (p == lo || bc[(size_t)*p] != bc[(size_t)p[-1]]) ++cnt;
    nblk[(size_t)i] = cnt;
  }
  std::vector<int32_t> rowptr((size_t)nbrows + 1, 0);
  int64_t nnzb = 0;
  for (int32_t i = 0; i < nbrows; ++i) { nnzb += nblk[(size_t)i]; rowptr[(size_t)i + 1] = (int32_t)nnzb; }
  if (nnzb * bs_r * bs_c >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "the assembled matrix has 2^31 or more values");
  std::vector<int32_t> colidx((size_t)nnzb), segptr((size_t)nnzb + 1);
  segptr[(size_t)nnzb] = (int32_t)nkept;
#pragma omp parallel for schedule(dynamic, 1024)
  for (int32_t i = 0; i < nbrows; ++i) {
    int32_t s = rowptr[(size_t)i];
    for (int64_t p = rstart[(size_t)i]; p < rstart[(size_t)i + 1]; ++p)
      if (p == rstart[(size_t)i] || bc[(size_t)byrow[(size_t)p]] != bc[(size_t)byrow[(size_t)p - 1]]) {
        colidx[(size_t)s] = bc[(size_t)byrow[(size_t)p]];
        segptr[(size_t)s] = (int32_t)p;
        ++s;
      }
  }
  // runs of destination blocks for the staged kernel: as many as fill one of its shared-memory buffers
  std::vector<int32_t> ctas;
  {
    const int32_t cap = BCOO_ITEMS / (bs_r * bs_c);
    bool fits = true;
    for (int64_t b0 = 0; b0 < nnzb && fits;) {
      int64_t b1 = b0;
      while (b1 < nnzb && b1 - b0 < BCOO_NBMAX && segptr[(size_t)b1 + 1] - segptr[(size_t)b0] <= cap) ++b1;
      if (b1 == b0) { fits = false; break; }   // one block with more contributions than a buffer parks
      ctas.push_back((int32_t)b0); ctas.push_back((int32_t)(b1 - b0));
      ctas.push_back(segptr[(size_t)b0]); ctas.push_back(segptr[(size_t)b1] - segptr[(size_t)b0]);
      b0 = b1;
    }
    if (!fits) ctas.clear();
  }
  if (!ctas.empty()) {   // cold: the staged kernel's shared memory, on the device the plan lives on
    cudaError_t e = cudaSuccess;
    switch (bs_r * bs_c) {
      case 4: e = cudaFuncSetAttribute(bcoo_flat_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BCOO_FLAT_SMEM); break;
      case 6: e = cudaFuncSetAttribute(bcoo_flat_kernel<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BCOO_FLAT_SMEM); break;
      case 9: e = cudaFuncSetAttribute(bcoo_flat_kernel<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BCOO_FLAT_SMEM); break;
      case 18: e = cudaFuncSetAttribute(bcoo_flat_kernel<18>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BCOO_FLAT_SMEM); break;
      case 36: e = cudaFuncSetAttribute(bcoo_flat_kernel<36>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BCOO_FLAT_SMEM); break;
      default: break;
    }
    if (e != cudaSuccess) return fail(BSR_ERR_CUDA, "bcoo_flat_kernel: cannot opt in to shared memory: %s", cudaGetErrorString(e));
  }
  bcoo_plan_s* pl = new (std::nothrow) bcoo_plan_s();
  if (!pl) return fail(BSR_ERR_ALLOC, "host allocation failed");
  pl->n = n; pl->nnzb = nnzb; pl->nbrows = nbrows; pl->nbcols = nbcols; pl->bs_r = bs_r; pl->bs_c = bs_c;
  pl->nctas = (int64_t)ctas.size() / 4;
  int rc = upload(&pl->rowptr, rowptr, st);
  if (rc == BSR_OK) rc = upload(&pl->colidx, colidx, st);
  if (rc == BSR_OK) rc = upload(&pl->segptr, segptr, st);
  if (rc == BSR_OK) rc = upload(&pl->perm, byrow, st);
  if (rc == BSR_OK && pl->nctas) rc = upload(&pl->ctas, ctas, st);
  if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  if (rc != BSR_OK) { bcoo_release(pl); return rc; }
  pl->magic = BCOO_MAGIC;
  if (nnzb_out) *nnzb_out = nnzb;
  *out = pl;
  return BSR_OK;
}

int bcoo_structure(bcoo_plan_t pl, int32_t* d_rowptr, int32_t* d_colidx, void* stream) {
  if (!pl || pl->magic != BCOO_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!d_rowptr || (pl->nnzb && !d_colidx)) return fail(BSR_ERR_NULL, "null output array");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemcpyAsync(d_rowptr, pl->rowptr, ((size_t)pl->nbrows + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (pl->nnzb) CUDA_TRY(cudaMemcpyAsync(d_colidx, pl->colidx, (size_t)pl->nnzb * 4, cudaMemcpyDeviceToDevice, st));
  return BSR_OK;
}

int bcoo_set_values(bcoo_plan_t pl, const double* d_stream, double* d_vals, void* stream) {
  if (!pl || pl->magic != BCOO_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (pl->nnzb == 0) return BSR_OK;
  if (!d_stream || !d_vals) return fail(BSR_ERR_NULL, "null array");
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv("bcoo_set_values");
  const int bb = pl->bs_r * pl->bs_c;
  const int64_t nvals = pl->nnzb * bb;
  if (pl->nctas) {
    const int4* runs = reinterpret_cast<const int4*>(pl->ctas);
#define BCOO_FLAT(BB)                                                                                                 \
  case BB: {                                                                                                          \
    LAUNCH(bcoo_flat_kernel<BB>, (unsigned)pl->nctas, BCOO_THREADS, BCOO_FLAT_SMEM, st, runs, pl->segptr, pl->perm, d_stream, d_vals); \
    return BSR_OK;                                                                                                    \
  }
    switch (bb) {
      BCOO_FLAT(4) BCOO_FLAT(6) BCOO_FLAT(9) BCOO_FLAT(18) BCOO_FLAT(36)
      default: return fail(BSR_ERR_BLOCK, "unsupported block shape");
    }
#undef BCOO_FLAT
  }
  const unsigned grid = (unsigned)((nvals + 255) / 256);
  switch (bb) {
    case 4: LAUNCH(bcoo_sum_kernel<4>, grid, 256, 0, st, nvals, pl->segptr, pl->perm, d_stream, d_vals); break;
    case 6: LAUNCH(bcoo_sum_kernel<6>, grid, 256, 0, st, nvals, pl->segptr, pl->perm, d_stream, d_vals); break;
    case 9: LAUNCH(bcoo_sum_kernel<9>, grid, 256, 0, st, nvals, pl->segptr, pl->perm, d_stream, d_vals); break;
    case 18: LAUNCH(bcoo_sum_kernel<18>, grid, 256, 0, st, nvals, pl->segptr, pl->perm, d_stream, d_vals); break;
    case 36: LAUNCH(bcoo_sum_kernel<36>, grid, 256, 0, st, nvals, pl->segptr, pl->perm, d_stream, d_vals); break;
    default: return fail(BSR_ERR_BLOCK, "unsupported block shape");
  }
  return BSR_OK;
}

int bcoo_get_info(bcoo_plan_t pl, int64_t* n_contrib, int64_t* nnzb, int64_t* algorithmic_bytes) {
  if (!pl || pl->magic != BCOO_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (n_contrib) *n_contrib = pl->n;
  if (nnzb) *nnzb = pl->nnzb;
  // the value stream read once, the destination values written once, one stream position per contribution and one
  // segment pointer per destination block
  if (algorithmic_bytes)
    *algorithmic_bytes = 8LL * pl->bs_r * pl->bs_c * (pl->n + pl->nnzb) + 4LL * pl->n + 4LL * (pl->nnzb + 1);
  return BSR_OK;
}

int bcoo_destroy(bcoo_plan_t pl) {
  if (!pl) return BSR_OK;
  if (pl->magic != BCOO_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  bcoo_release(pl);
  return BSR_OK;
}

int bsr_gather_blocks(int64_t n, const int32_t* d_idx, int32_t bs, const double* d_src, double* d_dst, void* stream) {
  if (n < 0 || bs < 1) return fail(BSR_ERR_SHAPE, "bsr_gather_blocks: bad size");
  if (n == 0) return BSR_OK;
  if (!d_idx || !d_src || !d_dst) return fail(BSR_ERR_NULL, "bsr_gather_blocks: null array");
  const int64_t nvals = n * bs;
  if ((nvals + 255) / 256 >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "too many values for one launch");
  LAUNCH(gather_blocks_kernel, (unsigned)((nvals + 255) / 256), 256, 0, (cudaStream_t)stream, nvals, (int)bs, d_idx, d_src, d_dst);
  return BSR_OK;
}

int bsr_scatter_add_blocks(int64_t n, const int32_t* d_idx, int32_t bs, const double* d_src, double* d_dst, void* stream) {
  if (n < 0 || bs < 1) return fail(BSR_ERR_SHAPE, "bsr_scatter_add_blocks: bad size");
  if (n == 0) return BSR_OK;
  if (!d_idx || !d_src || !d_dst) return fail(BSR_ERR_NULL, "bsr_scatter_add_blocks: null array");
  const int64_t nvals = n * bs;
  if ((nvals + 255) / 256 >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "too many values for one launch");
  LAUNCH(scatter_add_blocks_kernel, (unsigned)((nvals + 255) / 256), 256, 0, (cudaStream_t)stream, nvals, (int)bs, d_idx, d_src, d_dst);
  return BSR_OK;
}

int fem_q1_element_coords(int32_t d, int32_t ne, int64_t e0, int64_t e1, int32_t* d_brow, int32_t* d_bcol, void* stream) {
  if ((d != 2 && d != 3) || ne < 1 || e0 < 0 || e1 < e0) return fail(BSR_ERR_SHAPE, "fem_q1_element_coords: bad argument");
  const int64_t nel = (d == 3) ? (int64_t)ne * ne * ne : (int64_t)ne * ne;
  if (e1 > nel) return fail(BSR_ERR_SHAPE, "element range outside the grid");
  const int64_t nc = (e1 - e0) << (2 * d);
  if (nc == 0) return BSR_OK;
  if (!d_brow || !d_bcol) return fail(BSR_ERR_NULL, "null coordinate array");
  if (nc >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "2^31 or more contributions");
  LAUNCH(q1_coords_kernel, (unsigned)((nc + 255) / 256), 256, 0, (cudaStream_t)stream, d, ne, e0, nc, d_brow, d_bcol);
  return BSR_OK;
}

int fem_q1_element_blocks(int32_t d, int32_t ne, int64_t e0, int64_t e1, const double* d_Ke, const double* d_E,
                          int32_t dirichlet, double* d_stream, void* stream) {
  if ((d != 2 && d != 3) || ne < 1 || e0 < 0 || e1 < e0) return fail(BSR_ERR_SHAPE, "fem_q1_element_blocks: bad argument");
  const int64_t nel = (d == 3) ? (int64_t)ne * ne * ne : (int64_t)ne * ne;
  if (e1 > nel) return fail(BSR_ERR_SHAPE, "element range outside the grid");
  const int64_t nc = (e1 - e0) << (2 * d);
  if (nc == 0) return BSR_OK;
  if (!d_Ke || !d_stream) return fail(BSR_ERR_NULL, "null array");
  const int64_t nblocks = (nc + 255) / 256;
  if (nblocks >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "stream too long for one launch");
  if (d == 3) LAUNCH(q1_blocks_kernel<3>, (unsigned)nblocks, 256, 0, (cudaStream_t)stream, ne, e0, nc, d_Ke, d_E, dirichlet, d_stream);
  else LAUNCH(q1_blocks_kernel<2>, (unsigned)nblocks, 256, 0, (cudaStream_t)stream, ne, e0, nc, d_Ke, d_E, dirichlet, d_stream);
  return BSR_OK;
}

}  // extern "C"
