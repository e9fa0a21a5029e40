// bsr.cu -- the block-CSR container, the blocked SpMV family and the cached explicit transpose.
//
// Container: PAPER.md:20-28, 62-66 (block-CSR with independent bs_r x bs_c).  SpMV: PAPER.md:22, 121, 140-147
// (bandwidth-bound; 8*bs_r*bs_c + 4 bytes per block).  Transpose cache: PAPER.md:103 ("the transpose R", rebuilt
// only when the prolongator's state changes).
//
// SpMV kernel design (sm_100a, HBM-bound, no tensor cores -- DESIGN.md "Kernels"):
//   A lane GROUP of LB lanes owns one stored block per step.  A block is a flat run of bs_r*bs_c doubles; when that
//   count is even a lane loads one 16-byte pair of the run (3x6, 6x3, 6x6, 2x2, 2x3, 3x2), otherwise one double (3x3,
//   whose 72-byte blocks are only 8-byte aligned).  Consecutive lanes read consecutive addresses, so a group's load
//   is one contiguous block and the GPW = 32/LB groups of a warp read GPW consecutive blocks (TEAM mode, long rows:
//   the whole warp on one block row) or GPW different block rows (ROW mode, short rows such as the prolongator's).
//   All index / value / x loads of U steps are issued before the first FMA.  The row sum is finished with warp
//   shuffles in a fixed order (deterministic); the epilogue (y = Ax, b - Ax, y -= Ax, y += Ax) is fused in.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include <mutex>
#include <unordered_set>

#include "internal.h"

namespace bsramg {

thread_local std::string t_err = "";
std::atomic<int64_t> g_launches{0};
std::atomic<int64_t> g_allocs{0};

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  t_err = buf;
  return code;
}

// library workspace: through the caller's allocator when one is registered (bsr_set_allocator), else cudaMalloc.
// Memory obtained from one source is returned to the same source.
static bsr_alloc_fn g_alloc = nullptr;
static bsr_free_fn g_free = nullptr;
static void* g_alloc_ctx = nullptr;
static std::mutex g_alloc_mu;
static std::unordered_set<void*> g_from_caller;

int dev_alloc(void** p, size_t bytes) {
  *p = nullptr;
  bsr_alloc_fn af;
  void* ctx;
  { std::lock_guard<std::mutex> lk(g_alloc_mu); af = g_alloc; ctx = g_alloc_ctx; }
  if (af) {
    void* q = af(bytes ? bytes : 16, ctx);
    if (!q) return fail(BSR_ERR_ALLOC, "the caller's allocator returned null for %zu bytes", bytes);
    if ((uintptr_t)q & 255) { return fail(BSR_ERR_ALIGN, "the caller's allocator returned memory that is not 256-byte aligned"); }
    { std::lock_guard<std::mutex> lk(g_alloc_mu); g_from_caller.insert(q); }
    *p = q;
    g_allocs.fetch_add(1, std::memory_order_relaxed);
    return BSR_OK;
  }
  cudaError_t e = cudaMalloc(p, bytes ? bytes : 16);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(e == cudaErrorMemoryAllocation ? BSR_ERR_ALLOC : BSR_ERR_CUDA, "cudaMalloc(%zu): %s", bytes,
                cudaGetErrorString(e));
  }
  g_allocs.fetch_add(1, std::memory_order_relaxed);
  return BSR_OK;
}
void dev_free(void* p) {
  if (!p) return;
  bsr_free_fn ff = nullptr;
  void* ctx = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_alloc_mu);
    auto it = g_from_caller.find(p);
    if (it != g_from_caller.end()) { g_from_caller.erase(it); ff = g_free; ctx = g_alloc_ctx; if (!ff) return; }
  }
  if (ff) ff(p, ctx);
  else cudaFree(p);
}

// ------------------------------------------------------------------ lane mapping of one block shape
// A stored block is a flat run of BB = BR*BC doubles.  When BB is even a lane owns the 16-byte pair (2q, 2q+1) of
// that run (PAIR); when BC is even too both elements sit in one block row and the matching x entries are one
// aligned 16-byte pair (ROWPAIR).  3x3 (72-byte blocks, only 8-byte aligned for odd k) uses one lane per element.
template <int BR, int BC>
struct Shape {
  static constexpr int BB = BR * BC;
  static constexpr bool PAIR = (BB % 2 == 0);
  static constexpr bool ROWPAIR = PAIR && (BC % 2 == 0);
  static constexpr int LB = PAIR ? BB / 2 : BB;            // lanes per block
  static constexpr int LPR = ROWPAIR ? BC / 2 : BC;        // lanes per block row (ROWPAIR and scalar layouts)
  static constexpr int GPW = 32 / LB;                      // lane groups per warp
};

// y (op)= A x.  TEAM = number of lane groups that share one block row (1 or GPW).  U = blocks in flight per group.
// Loads are unconditional (the block index is clamped to the row's last block, the product of a clamped step is
// discarded) so that all U index, value and x loads of a step are issued before the first FMA.
// MINB = resident CTAs per SM the register allocation is held to: stating it at all makes ptxas keep the batched loads;
// 6 (40 registers, 48 warps per SM) is best for rows of a few steps (A, P), 4 (56 registers) for long rows (R) --
// measured, profiles/r1f_staged_ptap.md.
template <int BR, int BC, int TEAM, int U, int EPI, int MINB, int RB>
__global__ void __launch_bounds__(256, MINB)
spmv_kernel(int32_t nbrows, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
            const double* __restrict__ vals, const double* __restrict__ x, double* __restrict__ y,
            const double* __restrict__ b) {
  using S = Shape<BR, BC>;
  constexpr int ROWS_PER_WARP = S::GPW / TEAM;
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int g = lane / S::LB;  // lane group
  const int q = lane % S::LB;  // lane inside the group
  const int team = g / TEAM, member = g % TEAM;
  const bool glive = g < ROWS_PER_WARP * TEAM;
  // element(s) of the block this lane owns
  const int eA = S::PAIR ? 2 * q : q;
  const int cA = eA % BC;
  const int cB = (eA + 1) % BC;  // PAIR && !ROWPAIR only
  // A warp takes RB consecutive row groups; their row pointers come in with ONE load per lane, so only the first
  // group of a warp pays the rowptr -> values dependency with a cold row pointer.
  static_assert(RB * ROWS_PER_WARP + 1 <= 32, "row pointers of a batch must fit one load per lane");
  const int64_t row_first = warp * (RB * ROWS_PER_WARP);
  if (row_first >= nbrows) return;  // warp-uniform
  const int32_t rp_lane = __ldg(rowptr + min(row_first + lane, (int64_t)nbrows));
#pragma unroll 1
  for (int j = 0; j < RB; ++j) {
  const int ri = j * ROWS_PER_WARP + (glive ? team : 0);
  const int64_t row = row_first + ri;
  const bool live = glive && (row < nbrows);
  const int32_t k0 = __shfl_sync(0xffffffffu, rp_lane, ri), k1 = __shfl_sync(0xffffffffu, rp_lane, ri + 1);
  // the lane that will write y[row * BR + r].  What its epilogue reads (b or the old y) is requested from DRAM BEFORE
  // the row's blocks, as an L2 prefetch, and loaded after them, ahead of the reduction's shuffles.  Measured on the 96^3
  // operator (plain y = A x: 0.340 ms): load after the reduction 0.398 / 0.403 (RESID / SUB); this 0.376 / 0.377; the
  // operand held in a register across the loop 0.379 / 0.425 (two of the 40 registers the batched loads live on);
  // that with 5 resident CTAs instead of 6 0.401 / 0.420.
  const int r = (S::PAIR && !S::ROWPAIR) ? q : q / S::LPR;
  const bool writer = live && member == 0 && ((S::PAIR && !S::ROWPAIR) ? (q < BR) : (q % S::LPR) == 0);
  if (EPI != EPI_ASSIGN && writer)
    asm volatile("prefetch.global.L2 [%0];" ::"l"((EPI == EPI_RESID ? b : y) + row * BR + r));
  double accA = 0.0, accB = 0.0;
  if (live) {
    for (int32_t k = k0 + member; k < k1; k += TEAM * U) {
      bool ok[U];
      int32_t kc[U], col[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int32_t ku = k + u * TEAM;
        ok[u] = ku < k1;
        kc[u] = ok[u] ? ku : k1 - 1;
        col[u] = __ldg(colidx + kc[u]);
      }
      if (S::ROWPAIR) {
        double2 v[U], xv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) v[u] = __ldcs(reinterpret_cast<const double2*>(vals + (int64_t)kc[u] * S::BB + eA));
#pragma unroll
        for (int u = 0; u < U; ++u) xv[u] = __ldg(reinterpret_cast<const double2*>(x + (int64_t)col[u] * BC + cA));
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const double t = fma(v[u].y, xv[u].y, v[u].x * xv[u].x);
          accA += ok[u] ? t : 0.0;
        }
      } else if (S::PAIR) {
        double2 v[U];
        double xa[U], xb[U];
#pragma unroll
        for (int u = 0; u < U; ++u) v[u] = __ldcs(reinterpret_cast<const double2*>(vals + (int64_t)kc[u] * S::BB + eA));
#pragma unroll
        for (int u = 0; u < U; ++u) {
          xa[u] = __ldg(x + (int64_t)col[u] * BC + cA);
          xb[u] = __ldg(x + (int64_t)col[u] * BC + cB);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          accA = fma(ok[u] ? v[u].x : 0.0, xa[u], accA);
          accB = fma(ok[u] ? v[u].y : 0.0, xb[u], accB);
        }
      } else {
        double v[U], xv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) v[u] = __ldcs(vals + (int64_t)kc[u] * S::BB + eA);
#pragma unroll
        for (int u = 0; u < U; ++u) xv[u] = __ldg(x + (int64_t)col[u] * BC + cA);
#pragma unroll
        for (int u = 0; u < U; ++u) accA = fma(ok[u] ? v[u] : 0.0, xv[u], accA);
      }
    }
  }
  // the epilogue's operand: an L2 hit by now, issued ahead of the reduction's shuffles
  double prev = 0.0;
  if (EPI != EPI_ASSIGN && writer) prev = (EPI == EPI_RESID) ? __ldg(b + row * BR + r) : y[row * BR + r];
  // 1) the TEAM groups of a row (lanes LB apart), fixed order
#pragma unroll
  for (int s = 1; s < TEAM; s <<= 1) {
    const double tA = __shfl_down_sync(0xffffffffu, accA, (s * S::LB) & 31);
    const double tB = __shfl_down_sync(0xffffffffu, accB, (s * S::LB) & 31);
    if (member + s < TEAM) { accA += tA; accB += tB; }
  }
  // 2) the lanes of one block row
  double out;
  if (S::PAIR && !S::ROWPAIR) {
    // lane t < BR of the group gathers elements t*BC .. t*BC+BC-1: element e sits in lane e/2, slot e%2
    out = 0.0;
    const int base = lane - q;
#pragma unroll
    for (int c = 0; c < BC; ++c) {
      const int e = (q < BR ? q : 0) * BC + c;
      const double a = __shfl_sync(0xffffffffu, accA, (base + e / 2) & 31);
      const double bb = __shfl_sync(0xffffffffu, accB, (base + e / 2) & 31);
      out += (e & 1) ? bb : a;
    }
  } else {
    out = accA;
    if (S::LPR == 3) {
      const double t1 = __shfl_down_sync(0xffffffffu, out, 1);
      const double t2 = __shfl_down_sync(0xffffffffu, out, 2);
      out = (out + t1) + t2;
    } else if (S::LPR == 2) {
      out += __shfl_down_sync(0xffffffffu, out, 1);
    }
  }
  if (writer) {
    const int64_t o = row * BR + r;
    if (EPI == EPI_ASSIGN) y[o] = out;
    else if (EPI == EPI_ADD) y[o] = prev + out;
    else y[o] = prev - out;
  }
  }  // batch of row groups
}

template <int BR, int BC, int TEAM, int U, int MINB, int RB>
static int spmv_dispatch_epi(bsr_t A, const double* x, double* y, const double* b, Epilogue epi, cudaStream_t st) {
  using S = Shape<BR, BC>;
  constexpr int ROWS_PER_WARP = (S::GPW / TEAM) * RB;
  const int64_t warps = ((int64_t)A->nbrows + ROWS_PER_WARP - 1) / ROWS_PER_WARP;
  const int64_t blocks = (warps + 7) / 8;
  if (blocks == 0) return BSR_OK;
  if (blocks > 0x7fffffffLL) return fail(BSR_ERR_LIMIT, "grid too large");
  const dim3 grid((unsigned)blocks), block(256);
  switch (epi) {
    case EPI_ASSIGN:
      LAUNCH((spmv_kernel<BR, BC, TEAM, U, EPI_ASSIGN, MINB, RB>), grid, block, 0, st, A->nbrows, A->d_rowptr, A->d_colidx,
             A->d_vals, x, y, b);
      break;
    case EPI_RESID:
    case EPI_SUB:
      return fail(BSR_ERR_SHAPE, "spmv: the subtracting epilogues were retired (vcycle.cu forms r = b - t itself)");
    default:
      LAUNCH((spmv_kernel<BR, BC, TEAM, U, EPI_ADD, MINB, RB>), grid, block, 0, st, A->nbrows, A->d_rowptr, A->d_colidx,
             A->d_vals, x, y, b);
      break;
  }
  return BSR_OK;
}

// ------------------------------------------------------------------ short rows: flat value stream (ROWPAIR shapes)
// Rows of a handful of blocks (the prolongator: 1-8 blocks of 3x6) leave the row-per-lane-group kernel waiting on the
// chain rowptr -> (colidx, values) -> x for every three rows.  Here a CTA takes FLAT_ROWS consecutive block rows, whose
// values are ONE contiguous run: every thread streams 16-byte pairs of that run (perfectly coalesced, no clamped
// steps, loads independent of the row pointers), multiplies by the matching x pair and parks the partial product in
// shared memory; then one thread per output entry adds its row's partials in a fixed order (block by block, pair by
// pair) and applies the epilogue.  Deterministic, no atomics.
// 64 rows per CTA, 4 loads in flight per thread, 6 resident CTAs: the best of the sweep in profiles/r1g_final.md
constexpr int FLAT_ROWS = 64;
constexpr int FLAT_THREADS = 256;
constexpr int FLAT_U = 4;
constexpr int FLAT_MINB = 6;

template <int BR, int BC, int EPI>
__global__ void __launch_bounds__(FLAT_THREADS, FLAT_MINB)
spmv_flat_kernel(int32_t nbrows, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
                 const double* __restrict__ vals, const double* __restrict__ x, double* __restrict__ y,
                 const double* __restrict__ b) {
  using S = Shape<BR, BC>;
  static_assert(S::ROWPAIR, "flat kernel needs 16-byte pairs inside one block row");
  constexpr int LB = S::LB, LPR = S::LPR;
  extern __shared__ __align__(16) unsigned char flat_smem[];
  int32_t* rp = reinterpret_cast<int32_t*>(flat_smem);                 // FLAT_ROWS + 1 row pointers
  double* part = reinterpret_cast<double*>(flat_smem + ((FLAT_ROWS + 1) * 4 + 15) / 16 * 16);
  const int tid = threadIdx.x;
  const int32_t r0 = blockIdx.x * FLAT_ROWS, r1 = min(r0 + FLAT_ROWS, nbrows);
  if (tid <= r1 - r0) rp[tid] = __ldg(rowptr + r0 + tid);
  const int32_t k0 = __ldg(rowptr + r0), k1 = __ldg(rowptr + r1);
  const int32_t T = (k1 - k0) * LB;                                    // 16-byte pairs of the CTA's run
  constexpr int NOUT = (FLAT_ROWS * BR + FLAT_THREADS - 1) / FLAT_THREADS;   // output entries per thread
  if (EPI != EPI_ASSIGN) {                                             // what the epilogue reads: on its way to L2
#pragma unroll
    for (int w = 0; w < NOUT; ++w) {
      const int o = tid + w * FLAT_THREADS;
      if (o < (r1 - r0) * BR) asm volatile("prefetch.global.L2 [%0];" ::"l"((EPI == EPI_RESID ? b : y) + (int64_t)r0 * BR + o));
    }
  }
  const double2* v2 = reinterpret_cast<const double2*>(vals) + (int64_t)k0 * LB;
  for (int32_t c = tid; c < T; c += FLAT_THREADS * FLAT_U) {
    int32_t cu[FLAT_U], col[FLAT_U];
    double2 v[FLAT_U], xv[FLAT_U];
#pragma unroll
    for (int u = 0; u < FLAT_U; ++u) {
      cu[u] = min(c + u * FLAT_THREADS, T - 1);                        // clamped: the tail repeats the last pair
      col[u] = __ldg(colidx + k0 + cu[u] / LB);
    }
#pragma unroll
    for (int u = 0; u < FLAT_U; ++u) v[u] = __ldcs(v2 + cu[u]);
#pragma unroll
    for (int u = 0; u < FLAT_U; ++u)
      xv[u] = __ldg(reinterpret_cast<const double2*>(x + (int64_t)col[u] * BC) + (cu[u] % LB) % LPR);
#pragma unroll
    for (int u = 0; u < FLAT_U; ++u)
      if (c + u * FLAT_THREADS < T) part[cu[u]] = fma(v[u].y, xv[u].y, v[u].x * xv[u].x);
  }
  __syncthreads();
#pragma unroll
  for (int w = 0; w < NOUT; ++w) {
    const int o = tid + w * FLAT_THREADS;
    if (o >= (r1 - r0) * BR) break;
    const int rl = o / BR, r = o - rl * BR;
    const int32_t ks = rp[rl] - k0, ke = rp[rl + 1] - k0;
    double sum = 0.0;
    for (int32_t kk = ks; kk < ke; ++kk) {
#pragma unroll
      for (int cv = 0; cv < LPR; ++cv) sum += part[kk * LB + r * LPR + cv];
    }
    const int64_t oi = (int64_t)r0 * BR + o;
    if (EPI == EPI_ASSIGN) y[oi] = sum;
    else if (EPI == EPI_RESID) y[oi] = __ldg(b + oi) - sum;
    else if (EPI == EPI_SUB) y[oi] = y[oi] - sum;
    else y[oi] = y[oi] + sum;
  }
}

// shared memory a CTA of the flat kernel may ask for (its partials; above that the row kernel runs instead)
constexpr int FLAT_SMEM_MAX = 100 * 1024;

// prepare = true (cold, from bsr_create): opts the four epilogue instantiations in to FLAT_SMEM_MAX bytes of dynamic
// shared memory on the current device; false: the hot launch
template <int BR, int BC>
static int spmv_flat_launch(bsr_t A, const double* x, double* y, const double* b, Epilogue epi, cudaStream_t st,
                            bool prepare = false) {
  using S = Shape<BR, BC>;
  const int64_t blocks = ((int64_t)A->nbrows + FLAT_ROWS - 1) / FLAT_ROWS;
  if (blocks == 0 && !prepare) return BSR_OK;
  const size_t smem = ((FLAT_ROWS + 1) * 4 + 15) / 16 * 16 + (size_t)A->flat_max_blocks * S::LB * 8;
  const dim3 grid((unsigned)blocks), block(FLAT_THREADS);
#define FLAT_CASE(E)                                                                                          \
  {                                                                                                           \
    auto kern = spmv_flat_kernel<BR, BC, E>;                                                                  \
    if (prepare) {                                                                                            \
      CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, FLAT_SMEM_MAX));       \
    } else {                                                                                                  \
      LAUNCH(kern, grid, block, smem, st, A->nbrows, A->d_rowptr, A->d_colidx, A->d_vals, x, y, b);           \
    }                                                                                                         \
  }
  if (prepare) {
    FLAT_CASE(EPI_ASSIGN) FLAT_CASE(EPI_ADD)
    return BSR_OK;
  }
  switch (epi) {
    case EPI_ASSIGN: FLAT_CASE(EPI_ASSIGN) break;
    case EPI_RESID:
    case EPI_SUB:
      return fail(BSR_ERR_SHAPE, "spmv: the subtracting epilogues were retired (vcycle.cu forms r = b - t itself)");
    default: FLAT_CASE(EPI_ADD) break;
  }
#undef FLAT_CASE
  return BSR_OK;
}

// row-kernel parameters frozen from the sweeps in profiles/r1i_end_of_round.md: 4 loads in flight in ROW mode; a warp
// takes 4 consecutive short rows per row-pointer load (6 resident CTAs), 1 long row (4 resident CTAs)
constexpr int SPMV_ROW_U = 4, SPMV_RB_LONG = 1, SPMV_RB = 4, SPMV_MINB_SHORT = 6;

template <int BR, int BC>
static bool spmv_uses_flat(bsr_t A) {
  using S = Shape<BR, BC>;
  if constexpr (S::ROWPAIR) return A->team_mode != 1 && !A->no_flat && ((FLAT_ROWS + 1) * 4 + 15) / 16 * 16 + (size_t)A->flat_max_blocks * S::LB * 8 <= (size_t)FLAT_SMEM_MAX;
  return false;
}

template <int BR, int BC>
static int spmv_dispatch_team(bsr_t A, const double* x, double* y, const double* b, Epilogue epi, cudaStream_t st) {
  using S = Shape<BR, BC>;
  if (A->team_mode == 1) {
    // the whole warp on one block row: U steps of GPW blocks cover a 27-block row of A in one pass
    constexpr int U = (S::GPW >= 8) ? 2 : (S::GPW == 1 ? 8 : 9);
    if (A->avg_row_len >= 2.0 * S::GPW * U) return spmv_dispatch_epi<BR, BC, S::GPW, U, 4, SPMV_RB_LONG>(A, x, y, b, epi, st);
    return spmv_dispatch_epi<BR, BC, S::GPW, U, SPMV_MINB_SHORT, SPMV_RB>(A, x, y, b, epi, st);
  }
  if constexpr (S::ROWPAIR) {
    // short rows of a pair-able shape: the flat stream kernel, if a CTA's partials fit in shared memory
    if (spmv_uses_flat<BR, BC>(A)) return spmv_flat_launch<BR, BC>(A, x, y, b, epi, st);
  }
  return spmv_dispatch_epi<BR, BC, 1, SPMV_ROW_U, 6, 1>(A, x, y, b, epi, st);
}

// cold (bsr_create / first transpose): opt the flat kernels of A's shape in to their shared memory on this device
template <int BR, int BC>
static int spmv_prepare_shape(bsr_t A) {
  if constexpr (Shape<BR, BC>::ROWPAIR) {
    if (spmv_uses_flat<BR, BC>(A)) return spmv_flat_launch<BR, BC>(A, nullptr, nullptr, nullptr, EPI_ASSIGN, 0, true);
  }
  return BSR_OK;
}
static int spmv_prepare(bsr_t A) {
#define PREP(BR, BC) return spmv_prepare_shape<BR, BC>(A)
  switch (A->bs_r * 10 + A->bs_c) {
    case 22: PREP(2, 2);
    case 23: PREP(2, 3);
    case 32: PREP(3, 2);
    case 33: PREP(3, 3);
    case 36: PREP(3, 6);
    case 63: PREP(6, 3);
    case 66: PREP(6, 6);
  }
#undef PREP
  return BSR_OK;
}

int spmv_launch(bsr_t A, const double* x, double* y, const double* b, Epilogue epi, cudaStream_t st) {
  if (((uintptr_t)x | (uintptr_t)y | (uintptr_t)b) & 15) return fail(BSR_ERR_ALIGN, "vector pointer not 16-byte aligned");
  const int key = A->bs_r * 10 + A->bs_c;
  switch (key) {
    case 22: return spmv_dispatch_team<2, 2>(A, x, y, b, epi, st);
    case 23: return spmv_dispatch_team<2, 3>(A, x, y, b, epi, st);
    case 32: return spmv_dispatch_team<3, 2>(A, x, y, b, epi, st);
    case 33: return spmv_dispatch_team<3, 3>(A, x, y, b, epi, st);
    case 36: return spmv_dispatch_team<3, 6>(A, x, y, b, epi, st);
    case 63: return spmv_dispatch_team<6, 3>(A, x, y, b, epi, st);
    case 66: return spmv_dispatch_team<6, 6>(A, x, y, b, epi, st);
  }
  return fail(BSR_ERR_BLOCK, "unsupported block shape %dx%d", A->bs_r, A->bs_c);
}

// ------------------------------------------------------------------ cached explicit transpose
void host_transpose_structure(int32_t nbrows, int32_t nbcols, const int32_t* rowptr, const int32_t* colidx,
                              std::vector<int32_t>& rowptr_t, std::vector<int32_t>& colidx_t,
                              std::vector<int32_t>& perm) {
  const int64_t nnzb = rowptr[nbrows];
  rowptr_t.assign((size_t)nbcols + 1, 0);
  colidx_t.resize((size_t)nnzb);
  perm.resize((size_t)nnzb);
  for (int64_t k = 0; k < nnzb; ++k) rowptr_t[(size_t)colidx[k] + 1]++;
  for (int32_t j = 0; j < nbcols; ++j) rowptr_t[(size_t)j + 1] += rowptr_t[j];
  std::vector<int32_t> fill(rowptr_t.begin(), rowptr_t.end() - 1);
  // rows visited in ascending order -> every transposed row comes out sorted by column
  for (int32_t i = 0; i < nbrows; ++i)
    for (int32_t k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      const int32_t t = fill[colidx[k]]++;
      colidx_t[t] = i;
      perm[t] = k;
    }
}

// T.vals[t] = (vals[perm[t]])^T ; one thread per value of T (coalesced writes)
__global__ void __launch_bounds__(256)
transpose_values_kernel(int64_t nvals, int br, int bc, const int32_t* __restrict__ perm,
                        const double* __restrict__ vals, double* __restrict__ tvals) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nvals) return;
  const int bb = br * bc;
  const int64_t t = e / bb;
  const int pos = (int)(e - t * bb);  // position in the bc x br transposed block
  const int c = pos / br, r = pos - c * br;
  tvals[e] = __ldg(vals + (int64_t)__ldg(perm + t) * bb + r * bc + c);
}

// most blocks any run of FLAT_ROWS consecutive rows (one CTA of the flat SpMV) holds
static int32_t flat_max_blocks_of(const std::vector<int32_t>& rp, int32_t nbrows) {
  int32_t mx = 0;
  for (int32_t r0 = 0; r0 < nbrows; r0 += FLAT_ROWS) mx = std::max(mx, rp[(size_t)std::min(r0 + FLAT_ROWS, nbrows)] - rp[(size_t)r0]);
  return mx;
}

static void choose_team_mode(bsr_t A) {
  // the whole warp shares a row only when the row keeps every lane group busy for several steps (rows of mixed
  // length around 2 steps -- the Q2 prolongator, 1-27 blocks -- do better one lane group per row: config 5
  // y = P x_c 0.121 -> 0.107 ms)
  int gpw = 1;
  switch (A->bs_r * 10 + A->bs_c) {
    case 22: gpw = 16; break;
    case 23: gpw = 10; break;
    case 32: gpw = 10; break;
    case 33: gpw = 3; break;
    case 36: gpw = 3; break;
    case 63: gpw = 3; break;
    default: gpw = 1;
  }
  A->team_mode = (A->avg_row_len >= 4.0 * gpw) ? 1 : 0;
}

int transpose_ensure(bsr_t A, cudaStream_t st) {
  if (!A->T) {  // cold: build the structure on the host from the mirror taken at bsr_create
    std::vector<int32_t> rp, ci, perm;
    host_transpose_structure(A->nbrows, A->nbcols, A->h_rowptr.data(), A->h_colidx.data(), rp, ci, perm);
    bsr_matrix_s* T = new (std::nothrow) bsr_matrix_s();
    if (!T) return fail(BSR_ERR_ALLOC, "host allocation failed");
    T->nbrows = A->nbcols; T->nbcols = A->nbrows; T->bs_r = A->bs_c; T->bs_c = A->bs_r; T->nnzb = A->nnzb;
    T->magic = BSR_MAGIC; T->owns_arrays = true;
    int32_t *d_rp = nullptr, *d_ci = nullptr;
    int rc = upload(&d_rp, rp, st);
    if (rc == BSR_OK) rc = upload(&d_ci, ci, st);
    if (rc == BSR_OK) rc = upload(&A->T_perm, perm, st);
    if (rc == BSR_OK) rc = dev_alloc_t(&T->d_vals, (size_t)A->nnzb * A->bs_r * A->bs_c);
    T->d_rowptr = d_rp; T->d_colidx = d_ci;
    if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "transpose upload failed");
    if (rc != BSR_OK) {
      dev_free(d_rp); dev_free(d_ci); dev_free(A->T_perm); dev_free(T->d_vals);
      A->T_perm = nullptr;
      delete T;
      return rc;
    }
    int32_t mx = 0;
    for (int32_t j = 0; j < T->nbrows; ++j) mx = std::max(mx, rp[(size_t)j + 1] - rp[j]);
    T->max_row_len = mx;
    T->avg_row_len = T->nbrows ? (double)T->nnzb / T->nbrows : 0.0;
    T->flat_max_blocks = flat_max_blocks_of(rp, T->nbrows);
    T->h_rowptr.swap(rp);
    T->h_colidx.swap(ci);
    choose_team_mode(T);
    if (spmv_prepare(T) != BSR_OK) T->no_flat = true;   // a device without the shared memory: row kernel
    A->T = T;
    A->T_state = -1;
  }
  if (A->T_state != A->state) {  // state gate: values re-transposed on the device only when A's values moved
    const int64_t nvals = A->nnzb * A->bs_r * A->bs_c;
    if (nvals > 0)
      LAUNCH(transpose_values_kernel, (unsigned)((nvals + 255) / 256), 256, 0, st, nvals, (int)A->bs_r, (int)A->bs_c,
             A->T_perm, A->d_vals, A->T->d_vals);
    A->T_state = A->state;
    A->T_builds++;
    A->T->state++;
  }
  return BSR_OK;
}

static bool valid(bsr_t A) { return A && A->magic == BSR_MAGIC; }

}  // namespace bsramg

using namespace bsramg;

// =================================================================== C ABI
extern "C" {

const char* bsr_last_error(void) { return t_err.c_str(); }

int bsr_set_allocator(bsr_alloc_fn alloc_fn, bsr_free_fn free_fn, void* ctx) {
  if ((alloc_fn == nullptr) != (free_fn == nullptr)) return fail(BSR_ERR_NULL, "bsr_set_allocator: give both functions or neither");
  std::lock_guard<std::mutex> lk(g_alloc_mu);
  g_alloc = alloc_fn; g_free = free_fn; g_alloc_ctx = ctx;
  return BSR_OK;
}

int bsr_counters(int64_t* n_kernel_launches, int64_t* n_allocs) {
  if (n_kernel_launches) *n_kernel_launches = g_launches.load();
  if (n_allocs) *n_allocs = g_allocs.load();
  return BSR_OK;
}

int bsr_create(bsr_t* out, int32_t nbrows, int32_t nbcols, int32_t bs_r, int32_t bs_c, int64_t nnzb,
               const int32_t* d_rowptr, const int32_t* d_colidx, double* d_vals, void* stream) {
  if (!out) return fail(BSR_ERR_NULL, "bsr_create: out is null");
  *out = nullptr;
  if (!d_rowptr || (nnzb > 0 && (!d_colidx || !d_vals))) return fail(BSR_ERR_NULL, "bsr_create: null array");
  if (nbrows < 0 || nbcols < 0 || nnzb < 0) return fail(BSR_ERR_SHAPE, "bsr_create: negative size");
  if (!shape_supported(bs_r, bs_c)) return fail(BSR_ERR_BLOCK, "unsupported block shape %dx%d", bs_r, bs_c);
  if (nnzb * bs_r * bs_c >= (1LL << 31)) return fail(BSR_ERR_LIMIT, "nnzb*bs_r*bs_c >= 2^31");
  if ((uintptr_t)d_vals & 15) return fail(BSR_ERR_ALIGN, "d_vals not 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  bsr_matrix_s* A = new (std::nothrow) bsr_matrix_s();
  if (!A) return fail(BSR_ERR_ALLOC, "host allocation failed");
  A->h_rowptr.resize((size_t)nbrows + 1);
  A->h_colidx.resize((size_t)nnzb);
  cudaError_t e = cudaMemcpyAsync(A->h_rowptr.data(), d_rowptr, ((size_t)nbrows + 1) * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && nnzb)
    e = cudaMemcpyAsync(A->h_colidx.data(), d_colidx, (size_t)nnzb * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) {
    delete A;
    cudaGetLastError();
    return fail(BSR_ERR_CUDA, "bsr_create: structure copy failed: %s", cudaGetErrorString(e));
  }
  // validation of the canonical form
  const int32_t* rp = A->h_rowptr.data();
  const int32_t* ci = A->h_colidx.data();
  int bad = 0;
  if (rp[0] != 0 || (int64_t)rp[nbrows] != nnzb) bad = 1;
  int32_t mx = 0;
  if (!bad) {
#pragma omp parallel for schedule(static) reduction(max : mx) reduction(| : bad)
    for (int32_t i = 0; i < nbrows; ++i) {
      const int32_t a = rp[i], b = rp[i + 1];
      if (b < a || a < 0 || (int64_t)b > nnzb) { bad |= 2; continue; }
      mx = std::max(mx, b - a);
      for (int32_t k = a; k < b; ++k) {
        if (ci[k] < 0 || ci[k] >= nbcols) bad |= 4;
        if (k > a && ci[k] <= ci[k - 1]) bad |= 8;
      }
    }
  }
  if (bad) {
    delete A;
    return fail(BSR_ERR_STRUCTURE, "malformed structure (%s%s%s%s)", (bad & 1) ? "rowptr ends " : "",
                (bad & 2) ? "rowptr not monotone " : "", (bad & 4) ? "column out of range " : "",
                (bad & 8) ? "columns not strictly ascending" : "");
  }
  A->nbrows = nbrows; A->nbcols = nbcols; A->bs_r = bs_r; A->bs_c = bs_c; A->nnzb = nnzb;
  A->d_rowptr = d_rowptr; A->d_colidx = d_colidx; A->d_vals = d_vals;
  A->magic = BSR_MAGIC;
  A->max_row_len = mx;
  A->avg_row_len = nbrows ? (double)nnzb / nbrows : 0.0;
  A->flat_max_blocks = flat_max_blocks_of(A->h_rowptr, nbrows);
  choose_team_mode(A);
  if (spmv_prepare(A) != BSR_OK) A->no_flat = true;   // no device yet / too little shared memory: row kernel
  *out = A;
  return BSR_OK;
}

int bsr_values_changed(bsr_t A) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  A->state++;
  return BSR_OK;
}

int bsr_rebind_values(bsr_t A, double* d_vals) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (!d_vals && A->nnzb > 0) return fail(BSR_ERR_NULL, "bsr_rebind_values: null array");
  if ((uintptr_t)d_vals & 15) return fail(BSR_ERR_ALIGN, "d_vals not 16-byte aligned");
  if (A->owns_arrays) return fail(BSR_ERR_PLAN, "library-owned matrix");
  A->d_vals = d_vals;
  A->state++;
  return BSR_OK;
}

int bsr_destroy(bsr_t A) {
  if (!A) return BSR_OK;
  if (A->magic != BSR_MAGIC) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A->T) {
    dev_free((void*)A->T->d_rowptr); dev_free((void*)A->T->d_colidx); dev_free(A->T->d_vals);
    A->T->magic = 0;
    delete A->T;
  }
  dev_free(A->T_perm);
  dev_free(A->stage_x); dev_free(A->stage_y);
  A->magic = 0;
  delete A;
  return BSR_OK;
}

int bsr_get_info(bsr_t A, int32_t* nbrows, int32_t* nbcols, int32_t* bs_r, int32_t* bs_c, int64_t* nnzb,
                 int64_t* state) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (nbrows) *nbrows = A->nbrows;
  if (nbcols) *nbcols = A->nbcols;
  if (bs_r) *bs_r = A->bs_r;
  if (bs_c) *bs_c = A->bs_c;
  if (nnzb) *nnzb = A->nnzb;
  if (state) *state = A->state;
  return BSR_OK;
}

int64_t bsr_spmv_bytes(bsr_t A) {
  if (!valid(A)) return -1;
  return A->nnzb * (8LL * A->bs_r * A->bs_c + 4) + 4LL * (A->nbrows + 1) + 8LL * A->bs_c * A->nbcols +
         8LL * A->bs_r * A->nbrows;
}

int bsr_spmv(bsr_t A, const double* d_x, double* d_y, void* stream) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A->nbrows == 0) return BSR_OK;  // nothing to write; null vectors are fine for an empty matrix
  if ((!d_x && A->nbcols > 0) || !d_y) return fail(BSR_ERR_NULL, "null vector");
  NvtxRange nv("bsr_spmv");
  return spmv_launch(A, d_x, d_y, nullptr, EPI_ASSIGN, (cudaStream_t)stream);
}

int bsr_transpose_prepare(bsr_t A, int64_t* n_value_builds, void* stream) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  BSR_TRY(transpose_ensure(A, (cudaStream_t)stream));
  if (n_value_builds) *n_value_builds = A->T_builds;
  return BSR_OK;
}

int bsr_spmv_t(bsr_t A, const double* d_x, double* d_y, void* stream) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (A->nbcols == 0) return BSR_OK;
  if ((!d_x && A->nbrows > 0) || !d_y) return fail(BSR_ERR_NULL, "null vector");
  NvtxRange nv("bsr_spmv_t");
  BSR_TRY(transpose_ensure(A, (cudaStream_t)stream));
  return spmv_launch(A->T, d_x, d_y, nullptr, EPI_ASSIGN, (cudaStream_t)stream);
}

int bsr_spmv_host(bsr_t A, int32_t trans, const double* h_x, double* h_y, void* stream) {
  if (!valid(A)) return fail(BSR_ERR_NULL, "invalid matrix handle");
  if (!h_x || !h_y) return fail(BSR_ERR_NULL, "null vector");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nx = (size_t)(trans ? A->nbrows * (int64_t)A->bs_r : A->nbcols * (int64_t)A->bs_c);
  const size_t ny = (size_t)(trans ? A->nbcols * (int64_t)A->bs_c : A->nbrows * (int64_t)A->bs_r);
  // staging vectors live on the handle: allocated at first use (cold), reused afterwards
  int rc = BSR_OK;
  if (A->stage_nx < nx) { dev_free(A->stage_x); A->stage_x = nullptr; A->stage_nx = 0; rc = dev_alloc_t(&A->stage_x, nx); if (rc == BSR_OK) A->stage_nx = nx; }
  if (rc == BSR_OK && A->stage_ny < ny) { dev_free(A->stage_y); A->stage_y = nullptr; A->stage_ny = 0; rc = dev_alloc_t(&A->stage_y, ny); if (rc == BSR_OK) A->stage_ny = ny; }
  double *dx = A->stage_x, *dy = A->stage_y;
  if (rc == BSR_OK && cudaMemcpyAsync(dx, h_x, nx * 8, cudaMemcpyHostToDevice, st) != cudaSuccess)
    rc = fail(BSR_ERR_CUDA, "H2D copy failed");
  if (rc == BSR_OK) rc = trans ? bsr_spmv_t(A, dx, dy, stream) : bsr_spmv(A, dx, dy, stream);
  if (rc == BSR_OK && cudaMemcpyAsync(h_y, dy, ny * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess)
    rc = fail(BSR_ERR_CUDA, "D2H copy failed");
  if (rc == BSR_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(BSR_ERR_CUDA, "stream synchronise failed");
  return rc;
}

}  // extern "C"
