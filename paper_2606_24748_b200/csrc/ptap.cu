// ptap.cu -- Galerkin product A_c = P^T A P: cold symbolic phase and the hot two-stage numeric recompute.
//
// PAPER.md:42, 58 (A_c = P^T A P); 80-83 (symbolic once, numeric per operator change, MAT_REUSE_MATRIX);
// 103 ("local blocked triple product", cached P-side data gated on P's state, no host round trip on reuse);
// 97-99, 248-250 (blocked COO plan: coordinates declared once, contiguous bs_r*bs_c runs summed per block);
// 219 (the dominant fine-level kernel is the numeric A*P with block sizes <3,3,6>).
//
// Numeric design: both stages are the same output-stationary block product
//     C(u) = sum_p X[xrow0 + ox[p]] * Y[ystart[xrow0 + ox[p]] + oy[p]]
// stage 1: X = A (bf x bf), Y = P (bf x bc), C = AP;  stage 2: X = R (bc x bf), Y = AP (bf x bc), C = A_c.
// One thread owns one output block: the M x N accumulator lives in registers, the products of the block are
// walked in the plan's fixed order (ascending inner index) and the block is written once.  No atomics, no
// zero-fill pass, bit-reproducible.
#include <algorithm>
#include <cstring>
#include <cstdlib>

#include "internal.h"
#include "ptap_stream.h"

struct ptap_plan_s {
  uint64_t magic = 0;
  bsr_t A = nullptr, P = nullptr;
  int64_t nnzb_a = 0, nnzb_p = 0;
  int32_t bf = 0, bc = 0, nbrows_a = 0, nbrows_c = 0;
  int64_t nnzb_ap = 0, nnzb_c = 0, nprod1 = 0, nprod2 = 0;
  bool wide1 = false, wide2 = false;  // pair offsets need 16 bits each
  int32_t *rowptr_ap = nullptr, *colidx_ap = nullptr, *rowidx_ap = nullptr, *pairptr1 = nullptr, *pstart = nullptr;
  int32_t *rowptr_c = nullptr, *colidx_c = nullptr, *rowidx_c = nullptr, *pairptr2 = nullptr, *apstart = nullptr;
  void *pairs1 = nullptr, *pairs2 = nullptr;
  double* vals_ap = nullptr;
  bsramg::StreamDev s1, s2;  // brick-staged schedules of the two stages (ok == false: gather kernels)
  // the chunked host-buffer path (ptap_numeric_host): a copy stream and events, created at its first use (cold)
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_main = nullptr, ev_copy[16] = {};
};
static const int HOST_CHUNKS_IN = 8, HOST_CHUNKS_OUT = 4;
static const uint64_t PLAN_MAGIC = 0x5054415031303030ull;

namespace bsramg {

template <int NE>
__device__ __forceinline__ void load_block(const double* __restrict__ p, double (&v)[NE]) {
  if (NE % 2 == 0) {
#pragma unroll
    for (int e = 0; e < NE / 2; ++e) {
      const double2 t = __ldg(reinterpret_cast<const double2*>(p) + e);
      v[2 * e] = t.x;
      v[2 * e + 1] = t.y;
    }
  } else {
#pragma unroll
    for (int e = 0; e < NE; ++e) v[e] = __ldg(p + e);
  }
}

template <int NE>
__device__ __forceinline__ void store_block(double* __restrict__ p, const double (&v)[NE]) {
  if (NE % 2 == 0) {
#pragma unroll
    for (int e = 0; e < NE / 2; ++e) reinterpret_cast<double2*>(p)[e] = make_double2(v[2 * e], v[2 * e + 1]);
  } else {
#pragma unroll
    for (int e = 0; e < NE; ++e) p[e] = v[e];
  }
}

template <typename PairT>
struct PairCode;
template <>
struct PairCode<uint16_t> {
  __device__ __forceinline__ static int x(uint16_t p) { return p & 0xff; }
  __device__ __forceinline__ static int y(uint16_t p) { return p >> 8; }
};
template <>
struct PairCode<uint32_t> {
  __device__ __forceinline__ static int x(uint32_t p) { return p & 0xffff; }
  __device__ __forceinline__ static int y(uint32_t p) { return p >> 16; }
};

// C (M x N blocks) = gathered sum of X (M x K) * Y (K x N); one thread per output block
template <int M, int K, int N, typename PairT>
__global__ void __launch_bounds__(128)
block_product_kernel(int32_t nout, const int32_t* __restrict__ rowidx, const int32_t* __restrict__ rowptr_x,
                     const int32_t* __restrict__ ystart, const int32_t* __restrict__ pairptr,
                     const PairT* __restrict__ pairs, const double* __restrict__ xvals,
                     const double* __restrict__ yvals, double* __restrict__ cvals) {
  const int32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= nout) return;
  const int32_t x0 = __ldg(rowptr_x + __ldg(rowidx + u));
  const int32_t p0 = __ldg(pairptr + u), p1 = __ldg(pairptr + u + 1);
  double acc[M * N];
#pragma unroll
  for (int e = 0; e < M * N; ++e) acc[e] = 0.0;
  for (int32_t p = p0; p < p1; ++p) {
    const PairT code = __ldg(pairs + p);
    const int32_t xs = x0 + PairCode<PairT>::x(code);
    const int32_t ys = __ldg(ystart + xs) + PairCode<PairT>::y(code);
    double xb[M * K], yb[K * N];
    load_block<M * K>(xvals + (int64_t)xs * (M * K), xb);
    load_block<K * N>(yvals + (int64_t)ys * (K * N), yb);
#pragma unroll
    for (int r = 0; r < M; ++r)
#pragma unroll
      for (int c = 0; c < N; ++c)
#pragma unroll
        for (int m = 0; m < K; ++m) acc[r * N + c] = fma(xb[r * K + m], yb[m * N + c], acc[r * N + c]);
  }
  store_block<M * N>(cvals + (int64_t)u * (M * N), acc);
}

template <int M, int K, int N>
static int product_launch(bool wide, int64_t nout, const int32_t* rowidx, const int32_t* rowptr_x,
                          const int32_t* ystart, const int32_t* pairptr, const void* pairs, const double* xvals,
                          const double* yvals, double* cvals, cudaStream_t st) {
  if (nout == 0) return BSR_OK;
  const unsigned grid = (unsigned)((nout + 127) / 128);
  if (wide)
    LAUNCH((block_product_kernel<M, K, N, uint32_t>), grid, 128, 0, st, (int32_t)nout, rowidx, rowptr_x, ystart,
           pairptr, (const uint32_t*)pairs, xvals, yvals, cvals);
  else
    LAUNCH((block_product_kernel<M, K, N, uint16_t>), grid, 128, 0, st, (int32_t)nout, rowidx, rowptr_x, ystart,
           pairptr, (const uint16_t*)pairs, xvals, yvals, cvals);
  return BSR_OK;
}

template <typename T>
static int stream_up(const std::vector<T>& h, const T** d, StreamDev& sd, cudaStream_t st) {
  T* p = nullptr;
  BSR_TRY(upload(&p, h, st));
  sd.owned.push_back(p);
  sd.bytes += (int64_t)h.size() * sizeof(T);
  *d = p;
  return BSR_OK;
}

int stream_upload(const StreamShape& sh, const StreamPlan& sp, StreamDev& sd, cudaStream_t st, bool smooth) {
  sd = StreamDev();
  if (!sp.ok) return BSR_OK;
  StreamArgs& a = sd.args;
  int rc = stream_up(sp.bricks, &a.bricks, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.chunks, &a.chunks, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.xruns, &a.xruns, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.yruns, &a.yruns, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.entries, &a.entries, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.passes, &a.passes, sd, st);
  if (rc == BSR_OK) rc = stream_up(sp.meta, &a.meta, sd, st);
  if (rc == BSR_OK)   // shared-memory opt-in of the kernel that will run this plan
    rc = smooth ? stream_launch_smooth(sh.M, sh.N, a, 0, sp.max_smem, st, true)
                : stream_launch(sh.M, sh.K, sh.N, a, sp.persist, 0, sp.max_smem, st, true);
  if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "stream plan upload failed");
  if (rc != BSR_OK) { stream_release(sd); return rc; }
  sd.ok = true; sd.persist = sp.persist; sd.nbricks = sp.nbricks(); sd.smem = sp.max_smem;
  sd.brick_maxrow_prefix = sp.brick_maxrow;
  for (size_t b = 1; b < sd.brick_maxrow_prefix.size(); ++b)
    sd.brick_maxrow_prefix[b] = std::max(sd.brick_maxrow_prefix[b], sd.brick_maxrow_prefix[b - 1]);
  if (sp.persist) {
    sd.brick_out_end.resize(sp.bricks.size());
    for (size_t b = 0; b < sp.bricks.size(); ++b) sd.brick_out_end[b] = sp.bricks[b].out + sp.bricks[b].nslots;
  }
  return BSR_OK;
}

void stream_release(StreamDev& sd) {
  for (void* p : sd.owned) dev_free(p);
  sd = StreamDev();
}

static int stage1(ptap_plan_t pl, cudaStream_t st) {
  bsr_t A = pl->A, P = pl->P;
  if (pl->s1.ok) {
    StreamArgs a = pl->s1.args;
    a.xvals = A->d_vals; a.yvals = P->d_vals; a.cvals = pl->vals_ap;
    return stream_launch(pl->bf, pl->bf, pl->bc, a, false, pl->s1.nbricks, pl->s1.smem, st);
  }
#define S1(BF, BC)                                                                                             \
  return product_launch<BF, BF, BC>(pl->wide1, pl->nnzb_ap, pl->rowidx_ap, A->d_rowptr, pl->pstart, pl->pairptr1, \
                                    pl->pairs1, A->d_vals, P->d_vals, pl->vals_ap, st)
  switch (pl->bf * 10 + pl->bc) {
    case 22: S1(2, 2);
    case 23: S1(2, 3);
    case 32: S1(3, 2);
    case 33: S1(3, 3);
    case 36: S1(3, 6);
    case 63: S1(6, 3);
    case 66: S1(6, 6);
  }
#undef S1
  return fail(BSR_ERR_BLOCK, "unsupported block shapes in PtAP");
}

static int stage2(ptap_plan_t pl, double* d_vals_c, cudaStream_t st) {
  bsr_t R = pl->P->T;
  if (pl->s2.ok) {
    StreamArgs a = pl->s2.args;
    a.xvals = R->d_vals; a.yvals = pl->vals_ap; a.cvals = d_vals_c;
    return stream_launch(pl->bc, pl->bf, pl->bc, a, true, pl->s2.nbricks, pl->s2.smem, st);
  }
#define S2(BF, BC)                                                                                              \
  return product_launch<BC, BF, BC>(pl->wide2, pl->nnzb_c, pl->rowidx_c, R->d_rowptr, pl->apstart, pl->pairptr2, \
                                    pl->pairs2, R->d_vals, pl->vals_ap, d_vals_c, st)
  switch (pl->bf * 10 + pl->bc) {
    case 22: S2(2, 2);
    case 23: S2(2, 3);
    case 32: S2(3, 2);
    case 33: S2(3, 3);
    case 36: S2(3, 6);
    case 63: S2(6, 3);
    case 66: S2(6, 6);
  }
#undef S2
  return fail(BSR_ERR_BLOCK, "unsupported block shapes in PtAP");
}

static bool plan_ok(ptap_plan_t pl) { return pl && pl->magic == PLAN_MAGIC; }

static int plan_check(ptap_plan_t pl, bsr_t A, bsr_t P) {
  if (!plan_ok(pl)) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!A || !P || A->magic != BSR_MAGIC || P->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A != pl->A || P != pl->P || A->nnzb != pl->nnzb_a || P->nnzb != pl->nnzb_p)
    return fail(BSR_ERR_PLAN, "plan was built from different matrices");
  return BSR_OK;
}

template <typename PairT>
static void pack_pairs(const std::vector<uint16_t>& ox, const std::vector<uint16_t>& oy, int shift,
                       std::vector<PairT>& out) {
  out.resize(ox.size());
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < (int64_t)ox.size(); ++p) out[(size_t)p] = (PairT)(ox[(size_t)p] | ((uint32_t)oy[(size_t)p] << shift));
}

static int upload_pairs(void** d, bool wide, const std::vector<uint16_t>& ox, const std::vector<uint16_t>& oy,
                        cudaStream_t st) {
  int rc;
  if (wide) {
    std::vector<uint32_t> packed;
    pack_pairs<uint32_t>(ox, oy, 16, packed);
    uint32_t* p = nullptr;
    rc = upload(&p, packed, st);
    *d = p;
    if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  } else {
    std::vector<uint16_t> packed;
    pack_pairs<uint16_t>(ox, oy, 8, packed);
    uint16_t* p = nullptr;
    rc = upload(&p, packed, st);
    *d = p;
    if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  }
  return rc;
}

static void plan_release(ptap_plan_t pl) {
  if (!pl) return;
  if (pl->copy_stream) cudaStreamDestroy(pl->copy_stream);
  if (pl->ev_main) cudaEventDestroy(pl->ev_main);
  for (cudaEvent_t e : pl->ev_copy) if (e) cudaEventDestroy(e);
  dev_free(pl->rowptr_ap); dev_free(pl->colidx_ap); dev_free(pl->rowidx_ap); dev_free(pl->pairptr1);
  dev_free(pl->pstart); dev_free(pl->rowptr_c); dev_free(pl->colidx_c); dev_free(pl->rowidx_c);
  dev_free(pl->pairptr2); dev_free(pl->apstart); dev_free(pl->pairs1); dev_free(pl->pairs2); dev_free(pl->vals_ap);
  stream_release(pl->s1); stream_release(pl->s2);
  pl->magic = 0;
  delete pl;
}

static int64_t bsr_bytes(int64_t nnzb, int br, int bc, int64_t nbrows) {
  return nnzb * (8LL * br * bc + 4) + 4LL * (nbrows + 1);
}

}  // namespace bsramg

namespace bsramg {
Options& options() {
  static Options o;
  return o;
}
}  // namespace bsramg

using namespace bsramg;

extern "C" {

int bsr_set_option(const char* name, int64_t value) {
  if (!name) return fail(BSR_ERR_NULL, "bsr_set_option: null name");
  Options& o = options();
  if (!strcmp(name, "ptap_force_gather")) o.force_gather = value != 0;
  else if (!strcmp(name, "ptap_smem_stage1") && value >= 4096) o.smem_stage1 = value;
  else if (!strcmp(name, "ptap_smem_stage2") && value >= 4096) o.smem_stage2 = value;
  else return fail(BSR_ERR_SHAPE, "bsr_set_option: unknown option or bad value '%s'", name);
  return BSR_OK;
}

int ptap_get_schedule(ptap_plan_t pl, int64_t* out8) {
  if (!pl || pl->magic != PLAN_MAGIC || !out8) return fail(BSR_ERR_NULL, "invalid plan handle");
  out8[0] = pl->s1.ok; out8[1] = pl->s1.nbricks; out8[2] = 0; out8[3] = pl->s1.smem;
  out8[4] = pl->s2.ok; out8[5] = pl->s2.nbricks; out8[6] = 0; out8[7] = pl->s2.smem;
  return BSR_OK;
}

int ptap_symbolic(ptap_plan_t* out, bsr_t A, bsr_t P, int32_t* nbrows_c, int64_t* nnzb_c, void* stream) {
  if (!out) return fail(BSR_ERR_NULL, "ptap_symbolic: out is null");
  *out = nullptr;
  if (!A || !P || A->magic != BSR_MAGIC || P->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A->nbrows != A->nbcols || A->bs_r != A->bs_c) return fail(BSR_ERR_SHAPE, "A must be square with square blocks");
  if (A->nbcols != P->nbrows || A->bs_c != P->bs_r)
    return fail(BSR_ERR_SHAPE, "A (%d block cols, bs %d) does not match P (%d block rows, bs_r %d)", A->nbcols,
                A->bs_c, P->nbrows, P->bs_r);
  if (!shape_supported(P->bs_c, P->bs_r) || !shape_supported(P->bs_c, P->bs_c))
    return fail(BSR_ERR_BLOCK, "unsupported block shapes in PtAP");
  cudaStream_t st = (cudaStream_t)stream;
  BSR_TRY(transpose_ensure(P, st));  // R = P^T, cached on P
  bsr_t R = P->T;
  HostPlan hp;
  int rc = hp.build(A->nbrows, A->h_rowptr.data(), A->h_colidx.data(), P->nbcols, P->h_rowptr.data(),
                    P->h_colidx.data(), R->h_rowptr.data(), R->h_colidx.data());
  if (rc != BSR_OK) return fail(rc, "ptap_symbolic: %s", hp.err.c_str());
  ptap_plan_s* pl = new (std::nothrow) ptap_plan_s();
  if (!pl) return fail(BSR_ERR_ALLOC, "host allocation failed");
  pl->A = A; pl->P = P; pl->nnzb_a = A->nnzb; pl->nnzb_p = P->nnzb;
  pl->bf = A->bs_r; pl->bc = P->bs_c; pl->nbrows_a = A->nbrows; pl->nbrows_c = P->nbcols;
  pl->nnzb_ap = (int64_t)hp.colidx_ap.size(); pl->nnzb_c = (int64_t)hp.colidx_c.size();
  pl->nprod1 = (int64_t)hp.k1.size(); pl->nprod2 = (int64_t)hp.t2.size();
  pl->wide1 = hp.max_k1 > 255 || hp.max_q1 > 255;
  pl->wide2 = hp.max_t2 > 255 || hp.max_s2 > 255;
  if (pl->nnzb_ap * pl->bf * pl->bc >= (1LL << 31) || pl->nnzb_c * pl->bc * pl->bc >= (1LL << 31)) {
    delete pl;
    return fail(BSR_ERR_LIMIT, "AP or A_c has 2^31 or more values");
  }
  const Options opt = options();
  rc = upload(&pl->rowptr_ap, hp.rowptr_ap, st);
  if (rc == BSR_OK) rc = upload(&pl->colidx_ap, hp.colidx_ap, st);
  if (rc == BSR_OK) rc = upload(&pl->rowptr_c, hp.rowptr_c, st);
  if (rc == BSR_OK) rc = upload(&pl->colidx_c, hp.colidx_c, st);
  if (rc == BSR_OK) rc = dev_alloc_t(&pl->vals_ap, (size_t)pl->nnzb_ap * pl->bf * pl->bc);
  if (rc == BSR_OK && !opt.force_gather) {
    // brick-staged schedules (ptap_stream.cpp); a stage whose shapes do not fit keeps the gather kernel
    std::vector<StreamBrickDef> bricks;
    StreamPlan sp;
    const StreamShape sh1{pl->bf, pl->bf, pl->bc}, sh2{pl->bc, pl->bf, pl->bc};
    stream_bricks_stage1(hp, sh1, opt.smem_stage1, A->h_rowptr.data(), A->h_colidx.data(), P->h_rowptr.data(), bricks);
    stream_build(sh1, STREAM_THREADS_DIRECT / 32, opt.smem_stage1, bricks, A->h_rowptr.data(), A->h_colidx.data(),
                 P->h_rowptr.data(), hp.rowptr_ap.data(), hp.pairptr1.data(), hp.k1.data(), hp.q1.data(), sp);
    rc = stream_upload(sh1, sp, pl->s1, st);
    if (rc == BSR_OK) {
      const int nw2 = STREAM_THREADS_PERSIST / 32;
      stream_bricks_stage2(hp, sh2, nw2, opt.smem_stage2, R->h_rowptr.data(), R->h_colidx.data(), bricks);
      stream_build(sh2, nw2, opt.smem_stage2, bricks, R->h_rowptr.data(), R->h_colidx.data(), hp.rowptr_ap.data(),
                   hp.rowptr_c.data(), hp.pairptr2.data(), hp.t2.data(), hp.s2.data(), sp);
      rc = stream_upload(sh2, sp, pl->s2, st);
    }
  }
  // the gather lists go to the device only for a stage that stays on the fallback kernels
  if (rc == BSR_OK && !pl->s1.ok) {
    rc = upload(&pl->rowidx_ap, hp.rowidx_ap, st);
    if (rc == BSR_OK) rc = upload(&pl->pairptr1, hp.pairptr1, st);
    if (rc == BSR_OK) rc = upload(&pl->pstart, hp.pstart, st);
    if (rc == BSR_OK) rc = upload_pairs(&pl->pairs1, pl->wide1, hp.k1, hp.q1, st);
  }
  if (rc == BSR_OK && !pl->s2.ok) {
    rc = upload(&pl->rowidx_c, hp.rowidx_c, st);
    if (rc == BSR_OK) rc = upload(&pl->pairptr2, hp.pairptr2, st);
    if (rc == BSR_OK) rc = upload(&pl->apstart, hp.apstart, st);
    if (rc == BSR_OK) rc = upload_pairs(&pl->pairs2, pl->wide2, hp.t2, hp.s2, st);
  }
  if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "plan upload failed");
  if (rc != BSR_OK) {
    plan_release(pl);
    return rc;
  }
  pl->magic = PLAN_MAGIC;
  if (nbrows_c) *nbrows_c = pl->nbrows_c;
  if (nnzb_c) *nnzb_c = pl->nnzb_c;
  *out = pl;
  return BSR_OK;
}

int ptap_structure(ptap_plan_t pl, int32_t* d_rowptr_c, int32_t* d_colidx_c, void* stream) {
  if (!plan_ok(pl)) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (!d_rowptr_c || (pl->nnzb_c && !d_colidx_c)) return fail(BSR_ERR_NULL, "null output array");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemcpyAsync(d_rowptr_c, pl->rowptr_c, ((size_t)pl->nbrows_c + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (pl->nnzb_c)
    CUDA_TRY(cudaMemcpyAsync(d_colidx_c, pl->colidx_c, (size_t)pl->nnzb_c * 4, cudaMemcpyDeviceToDevice, st));
  return BSR_OK;
}

int ptap_numeric_stage(ptap_plan_t pl, int32_t stage, bsr_t A, bsr_t P, double* d_vals_c, void* stream) {
  BSR_TRY(plan_check(pl, A, P));
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv(stage == 1 ? "ptap_numeric_stage1" : "ptap_numeric_stage2");
  if (stage == 1) return stage1(pl, st);
  if (stage == 2) {
    if (!d_vals_c && pl->nnzb_c) return fail(BSR_ERR_NULL, "d_vals_c is null");
    if ((uintptr_t)d_vals_c & 15) return fail(BSR_ERR_ALIGN, "d_vals_c must be 16-byte aligned");
    BSR_TRY(transpose_ensure(P, st));  // state gate: a no-op while P is untouched
    return stage2(pl, d_vals_c, st);
  }
  return fail(BSR_ERR_SHAPE, "stage must be 1 or 2");
}

int ptap_numeric(ptap_plan_t pl, bsr_t A, bsr_t P, double* d_vals_c, void* stream) {
  BSR_TRY(plan_check(pl, A, P));
  if (!d_vals_c && pl->nnzb_c) return fail(BSR_ERR_NULL, "d_vals_c is null");
  if ((uintptr_t)d_vals_c & 15) return fail(BSR_ERR_ALIGN, "d_vals_c must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  NvtxRange nv("ptap_numeric");
  BSR_TRY(transpose_ensure(P, st));  // state gate: re-transposes R's values only if P changed
  BSR_TRY(stage1(pl, st));
  return stage2(pl, d_vals_c, st);
}

int ptap_numeric_host(ptap_plan_t pl, bsr_t A, bsr_t P, const double* h_vals_a, double* h_vals_c, double* d_vals_c,
                      void* stream) {
  BSR_TRY(plan_check(pl, A, P));
  if (!h_vals_a || !h_vals_c || !d_vals_c) return fail(BSR_ERR_NULL, "null array");
  if ((uintptr_t)d_vals_c & 15) return fail(BSR_ERR_ALIGN, "d_vals_c must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t bba = (size_t)A->bs_r * A->bs_c * 8, bbc = (size_t)pl->bc * pl->bc * 8;
  if (!pl->s1.ok || !pl->s2.ok || pl->s1.nbricks < HOST_CHUNKS_IN || pl->s2.nbricks < HOST_CHUNKS_OUT) {
    // gather plans / tiny problems: copy, compute, copy
    CUDA_TRY(cudaMemcpyAsync(A->d_vals, h_vals_a, (size_t)A->nnzb * bba, cudaMemcpyHostToDevice, st));
    A->state++;
    BSR_TRY(ptap_numeric(pl, A, P, d_vals_c, stream));
    CUDA_TRY(cudaMemcpyAsync(h_vals_c, d_vals_c, (size_t)pl->nnzb_c * bbc, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return BSR_OK;
  }
  // staged plans: A's values arrive in row chunks on a copy stream; the bricks of stage 1 whose rows are complete are
  // launched behind each chunk, so AP = A*P hides under the transfer; A_c leaves in pieces behind stage 2 the same way
  if (!pl->copy_stream) {   // cold, once
    CUDA_TRY(cudaStreamCreateWithFlags(&pl->copy_stream, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_main, cudaEventDisableTiming));
    for (cudaEvent_t& e : pl->ev_copy) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  NvtxRange nv("ptap_numeric_host");
  cudaStream_t cs = pl->copy_stream;
  CUDA_TRY(cudaEventRecord(pl->ev_main, st));            // earlier work on `stream` may still read A's old values
  CUDA_TRY(cudaStreamWaitEvent(cs, pl->ev_main, 0));
  A->state++;
  BSR_TRY(transpose_ensure(P, st));                      // state gate
  const std::vector<int32_t>& rp = A->h_rowptr;
  const std::vector<int32_t>& need = pl->s1.brick_maxrow_prefix;
  int32_t row0 = 0;
  int64_t b0 = 0;
  for (int g = 0; g < HOST_CHUNKS_IN; ++g) {
    // rows [row0, row1): about 1/8 of the blocks each
    const int64_t target = A->nnzb * (g + 1) / HOST_CHUNKS_IN;
    int32_t row1 = (g + 1 == HOST_CHUNKS_IN) ? A->nbrows
                                             : (int32_t)(std::upper_bound(rp.begin(), rp.end(), (int32_t)target) - rp.begin() - 1);
    row1 = std::max(row1, row0);
    const size_t o0 = (size_t)rp[(size_t)row0] * bba, o1 = (size_t)rp[(size_t)row1] * bba;
    if (o1 > o0)
      CUDA_TRY(cudaMemcpyAsync((char*)A->d_vals + o0, (const char*)h_vals_a + o0, o1 - o0, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaEventRecord(pl->ev_copy[g], cs));
    CUDA_TRY(cudaStreamWaitEvent(st, pl->ev_copy[g], 0));
    // leading bricks that read no row at or beyond row1
    const int64_t b1 = (g + 1 == HOST_CHUNKS_IN)
                           ? pl->s1.nbricks
                           : (int64_t)(std::lower_bound(need.begin(), need.end(), row1) - need.begin());
    if (b1 > b0) {
      StreamArgs a = pl->s1.args;
      a.xvals = A->d_vals; a.yvals = P->d_vals; a.cvals = pl->vals_ap; a.brick0 = (int32_t)b0;
      BSR_TRY(stream_launch(pl->bf, pl->bf, pl->bc, a, false, b1 - b0, pl->s1.smem, st));
      b0 = b1;
    }
    row0 = row1;
  }
  // stage 2 in pieces; each piece's rows of A_c go home as soon as it is done
  bsr_t R = P->T;
  int64_t c0 = 0;
  size_t out0 = 0;
  for (int g = 0; g < HOST_CHUNKS_OUT; ++g) {
    const int64_t c1 = pl->s2.nbricks * (g + 1) / HOST_CHUNKS_OUT;
    if (c1 <= c0) continue;
    StreamArgs a = pl->s2.args;
    a.xvals = R->d_vals; a.yvals = pl->vals_ap; a.cvals = d_vals_c; a.brick0 = (int32_t)c0;
    BSR_TRY(stream_launch(pl->bc, pl->bf, pl->bc, a, true, c1 - c0, pl->s2.smem, st));
    CUDA_TRY(cudaEventRecord(pl->ev_copy[HOST_CHUNKS_IN + g], st));
    CUDA_TRY(cudaStreamWaitEvent(cs, pl->ev_copy[HOST_CHUNKS_IN + g], 0));
    const size_t out1 = (size_t)pl->s2.brick_out_end[(size_t)c1 - 1] * bbc;   // bricks write A_c in slot order
    if (out1 > out0)
      CUDA_TRY(cudaMemcpyAsync((char*)h_vals_c + out0, (const char*)d_vals_c + out0, out1 - out0, cudaMemcpyDeviceToHost, cs));
    out0 = out1;
    c0 = c1;
  }
  CUDA_TRY(cudaStreamSynchronize(cs));
  CUDA_TRY(cudaStreamSynchronize(st));
  return BSR_OK;
}

int ptap_get_info(ptap_plan_t pl, int64_t* nnzb_ap, int64_t* n_products_1, int64_t* n_products_2,
                  int64_t* algorithmic_bytes, int64_t* n_r_value_builds) {
  if (!plan_ok(pl)) return fail(BSR_ERR_NULL, "invalid plan handle");
  if (nnzb_ap) *nnzb_ap = pl->nnzb_ap;
  if (n_products_1) *n_products_1 = pl->nprod1;
  if (n_products_2) *n_products_2 = pl->nprod2;
  if (algorithmic_bytes) {
    const int64_t bA = bsr_bytes(pl->nnzb_a, pl->bf, pl->bf, pl->nbrows_a);
    const int64_t bP = bsr_bytes(pl->nnzb_p, pl->bf, pl->bc, pl->nbrows_a);
    const int64_t bR = bsr_bytes(pl->nnzb_p, pl->bc, pl->bf, pl->nbrows_c);
    const int64_t bAP = bsr_bytes(pl->nnzb_ap, pl->bf, pl->bc, pl->nbrows_a);
    const int64_t bC = bsr_bytes(pl->nnzb_c, pl->bc, pl->bc, pl->nbrows_c);
    *algorithmic_bytes = (bA + bP + bAP) + (bR + bAP + bC);
  }
  if (n_r_value_builds) *n_r_value_builds = pl->P->T_builds;
  return BSR_OK;
}

int ptap_get_ap(ptap_plan_t pl, int32_t* d_rowptr_ap, int32_t* d_colidx_ap, double* d_vals_ap, void* stream) {
  if (!plan_ok(pl)) return fail(BSR_ERR_NULL, "invalid plan handle");
  cudaStream_t st = (cudaStream_t)stream;
  if (d_rowptr_ap)
    CUDA_TRY(cudaMemcpyAsync(d_rowptr_ap, pl->rowptr_ap, ((size_t)pl->nbrows_a + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (d_colidx_ap && pl->nnzb_ap)
    CUDA_TRY(cudaMemcpyAsync(d_colidx_ap, pl->colidx_ap, (size_t)pl->nnzb_ap * 4, cudaMemcpyDeviceToDevice, st));
  if (d_vals_ap && pl->nnzb_ap)
    CUDA_TRY(cudaMemcpyAsync(d_vals_ap, pl->vals_ap, (size_t)pl->nnzb_ap * pl->bf * pl->bc * 8, cudaMemcpyDeviceToDevice, st));
  return BSR_OK;
}

int ptap_destroy(ptap_plan_t pl) {
  if (!pl) return BSR_OK;
  if (pl->magic != PLAN_MAGIC) return fail(BSR_ERR_NULL, "invalid plan handle");
  plan_release(pl);
  return BSR_OK;
}

}  // extern "C"
