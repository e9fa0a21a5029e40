// internal.h -- private declarations of libbsramg.so (not part of the C ABI; see include/bsr_amg.h).
#pragma once
#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include "bsr_amg.h"

namespace bsramg {

// ------------------------------------------------------------------ errors and counters
int fail(int code, const char* fmt, ...);
extern std::atomic<int64_t> g_launches;
extern std::atomic<int64_t> g_allocs;

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e__ = (expr);                                                                  \
    if (e__ != cudaSuccess) return ::bsramg::fail(BSR_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
  } while (0)

#define BSR_TRY(expr)            \
  do {                           \
    int rc__ = (expr);           \
    if (rc__ != BSR_OK) return rc__; \
  } while (0)

// every kernel launch of the library goes through this: counts it and checks the launch status
#define LAUNCH(kernel, grid, block, smem, stream, ...)                                   \
  do {                                                                                   \
    kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);                          \
    ::bsramg::g_launches.fetch_add(1, std::memory_order_relaxed);                        \
    cudaError_t e__ = cudaGetLastError();                                                \
    if (e__ != cudaSuccess) return ::bsramg::fail(BSR_ERR_CUDA, "launch %s: %s", #kernel, cudaGetErrorString(e__)); \
  } while (0)

// NVTX range around a hot entry point (tracing); a no-op unless a profiler is attached
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};

int dev_alloc(void** p, size_t bytes);  // cudaMalloc + counter (cold paths only)
void dev_free(void* p);

template <typename T>
int dev_alloc_t(T** p, size_t n) { return dev_alloc(reinterpret_cast<void**>(p), (n ? n : 1) * sizeof(T)); }

template <typename T>
int upload(T** d, const std::vector<T>& h, cudaStream_t st) {
  BSR_TRY(dev_alloc_t(d, h.size()));
  if (!h.empty()) CUDA_TRY(cudaMemcpyAsync(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st));
  return BSR_OK;
}

inline bool shape_supported(int br, int bc) {
  return (br == 2 && bc == 2) || (br == 2 && bc == 3) || (br == 3 && bc == 2) || (br == 3 && bc == 3) ||
         (br == 3 && bc == 6) || (br == 6 && bc == 3) || (br == 6 && bc == 6);
}

// epilogues of the SpMV kernels (the V-cycle glue fused into the product).  EPI_RESID / EPI_SUB
// (y = b - A x, y -= A x) are still understood by the kernels but no longer launched: at 10 % over the plain product
// they lost to subtracting inside the Chebyshev update (vcycle.cu); spmv_launch refuses them.
enum Epilogue { EPI_ASSIGN = 0, /* y = A x */ EPI_RESID = 1, EPI_SUB = 2, EPI_ADD = 3 /* y += A x */ };

// internal SpMV with epilogue (b: unused by the launched epilogues)
int spmv_launch(bsr_t A, const double* d_x, double* d_y, const double* d_b, Epilogue epi, cudaStream_t st);
// dinv[i] = inverse of A's bs x bs diagonal block of row i (point-block Jacobi data); *status |= 1 on a
// missing or singular block
int block_diag_inverse(bsr_t A, double* dinv, int* status, cudaStream_t st);
// C (m x n) = beta*C + alpha * A (m x k) * op(B), row-major, 128x128 tiles (dense_gemm.cu).  transB: B is n x k, else
// k x n.  batch problems at strides sA/sB/sC.  tri = 1: lower tiles only.  klim = 1: B lower triangular (k >= tile
// column start), 2: A lower triangular (k < tile row end).  koff: A is banded, row i has no nonzero left of column
// koff + i (very negative: none).  kcap: rows >= kcap of B are zero (0: none).  m, n multiples of 128, k of 16.
int dgemm128(bool transB, int m, int n, int k, double alpha, const double* A, int64_t lda, const double* B, int64_t ldb,
             double beta, double* C, int64_t ldc, int batch, int64_t sA, int64_t sB, int64_t sC, int tri, int klim,
             cudaStream_t st, int koff = -(1 << 30), int kcap = 0);
// makes sure the cached transpose exists and its values are current; hot when nothing changed
int transpose_ensure(bsr_t A, cudaStream_t st);

// ------------------------------------------------------------------ host side of the symbolic phase
struct HostPlan {
  // inputs (borrowed while build() runs)
  int32_t nbrows_a = 0, nbcols_p = 0;
  // structures
  std::vector<int32_t> rowptr_ap, colidx_ap, rowidx_ap;  // rowidx_ap[s] = fine row of AP slot s
  std::vector<int32_t> rowptr_c, colidx_c, rowidx_c;     // rowidx_c[u]  = coarse row of A_c slot u
  // stage 1: AP(s) = sum over p in [pairptr1[s], pairptr1[s+1]) of A(rowptr_a[i] + k1[p]) * P(pstart[...] + q1[p])
  std::vector<int32_t> pairptr1;
  std::vector<uint16_t> k1, q1;  // offsets inside A's row i / inside P's row j
  std::vector<int32_t> pstart;   // per A slot k: rowptr_p[colidx_a[k]]
  // stage 2: A_c(u) = sum over p of R(rowptr_r[I] + t2[p]) * AP(apstart[...] + s2[p])
  std::vector<int32_t> pairptr2;
  std::vector<uint16_t> t2, s2;  // offsets inside R's row I / inside AP's row i
  std::vector<int32_t> apstart;  // per R slot t: rowptr_ap[colidx_r[t]]
  int32_t max_k1 = 0, max_q1 = 0, max_t2 = 0, max_s2 = 0;
  std::string err;
  // stage 1 only (structure and gather lists of A*P): what prolongator smoothing needs (smooth.cu)
  int build_stage1(int32_t nbrows_a, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p,
                   const int32_t* rowptr_p, const int32_t* colidx_p);
  // builds everything from the host structures of A, P and R = P^T.  Returns BSR_OK or an error code.
  int build(int32_t nbrows_a, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p,
            const int32_t* rowptr_p, const int32_t* colidx_p, const int32_t* rowptr_r, const int32_t* colidx_r);
};

// explicit transpose structure on the host: R = P^T rows sorted; perm[t] = slot of P that R's slot t comes from
void host_transpose_structure(int32_t nbrows, int32_t nbcols, const int32_t* rowptr, const int32_t* colidx,
                              std::vector<int32_t>& rowptr_t, std::vector<int32_t>& colidx_t,
                              std::vector<int32_t>& perm);

// process-wide options of the COLD calls (bsr_set_option); never read by a hot call
struct Options {
  int64_t force_gather = 0;                 // 1: ptap_symbolic keeps the gather kernels (tests of the fallback)
  int64_t smem_stage1 = 112 * 1024;         // shared memory a stage-1 brick may use (two bricks per SM)
  int64_t smem_stage2 = 75000;              // stage 2: three coarse rows per SM (register-limited)
};
Options& options();

}  // namespace bsramg

// ------------------------------------------------------------------ the opaque handle types
struct bsr_matrix_s {
  int32_t nbrows = 0, nbcols = 0, bs_r = 0, bs_c = 0;
  int64_t nnzb = 0;
  const int32_t* d_rowptr = nullptr;
  const int32_t* d_colidx = nullptr;
  double* d_vals = nullptr;
  int64_t state = 0;  // bumped by bsr_values_changed
  uint64_t magic = 0;
  // host mirror of the structure (taken at bsr_create, used by the cold symbolic paths)
  std::vector<int32_t> h_rowptr, h_colidx;
  int32_t max_row_len = 0;
  double avg_row_len = 0;
  int team_mode = 0;  // 0: one lane group per row, 1: the whole warp per row
  int32_t flat_max_blocks = 0;  // most blocks in any run of 64 consecutive rows (flat SpMV shared-memory size)
  bool no_flat = false;         // the flat kernel's shared-memory opt-in failed at creation: use the row kernel
  // cached explicit transpose (library-owned)
  bsr_matrix_s* T = nullptr;
  int32_t* T_perm = nullptr;  // device: source slot per transposed slot
  int64_t T_state = -1;       // state of this matrix when T's values were last built
  int64_t T_builds = 0;
  bool owns_arrays = false;  // true for library-created matrices (the transposes)
  // staging vectors of the *_host convenience calls (allocated at first use, kept)
  double *stage_x = nullptr, *stage_y = nullptr;
  size_t stage_nx = 0, stage_ny = 0;
};
static const uint64_t BSR_MAGIC = 0x425352414d473031ull;

// ------------------------------------------------------------------ brick-staged block products (ptap_stream.cpp)
// One output-stationary block product C = X * Y (stage 1: X = A, Y = P; stage 2: X = R, Y = AP) cut into BRICKS
// (one CTA each) of CHUNKS.  A chunk stages a set of X row pieces and every Y row they reference in shared memory.
// A lane owns one output block C(row, slot) (M x N accumulators in registers).  A warp walks the X blocks of its
// row piece(s) in order ("k-synchronous"): at step k every lane of the row reads the same X block (a broadcast),
// and the lanes whose slot receives a product from X(row,k) -- bit `slot` of the block's MASK -- read consecutive
// blocks of Y's row (lane's block = rank of its bit in the mask), so shared-memory reads are broadcast or
// contiguous.  DIRECT bricks write each block once from registers at the end of a pass (stage 1).  PERSIST bricks
// keep the accumulators over all chunks, every warp taking a share of each chunk's X blocks, and add the warps'
// partial blocks in warp order through shared memory before writing the block once (stage 2) -- the atomic-free
// segmented scatter of SURVEY.md 8(a) a7.
namespace bsramg {

struct StreamEntry {   // 16 bytes: the lanes of one X row piece inside a pass, all in ONE window of the row's slots
  int32_t out;         // first C slot of the window (direct); unused (persist: the brick header carries it)
  int32_t xbase;       // staged X block index of the piece's first block
  int32_t mbase;       // staged meta index of the piece's first block FOR THIS WINDOW
  uint32_t packed;     // len (16 bits: X blocks = steps) | lane0 (5) | nslots-1 (5) | slot0 inside the window (5)
  static uint32_t pack(int len, int lane0, int nslots, int slot0) {
    return (uint32_t)len | ((uint32_t)lane0 << 16) | ((uint32_t)(nslots - 1) << 21) | ((uint32_t)slot0 << 26);
  }
  __host__ __device__ int len() const { return (int)(packed & 0xffffu); }
  __host__ __device__ int lane0() const { return (int)((packed >> 16) & 31u); }
  __host__ __device__ int nslots() const { return (int)((packed >> 21) & 31u) + 1; }
  __host__ __device__ int slot0() const { return (int)((packed >> 26) & 31u); }
};
struct StreamPass { int32_t e0, e1, steps, pad; };   // entries [e0, e1) (relative to the chunk), max len
struct StreamMeta { uint32_t mask, ybase; };          // per (staged X block, window): receiving slots of the window and
                                                      // the staged Y block of the first of them
struct StreamRun { int32_t src, n, dst; };            // copy n blocks from global block src to staged block dst
struct StreamBrickHdr { int32_t chunk0, nchunks, out, nslots; };   // out / nslots: persist bricks (C row of the brick)
struct StreamChunkHdr {   // 64 bytes: everything a CTA needs to know about a chunk, fetched with one load
  int64_t meta0;          // first staged X block in StreamPlan::meta
  int32_t nx, ny;         // staged X blocks and Y blocks
  int32_t ent0, nent, pass0, npass, xr0, nxr, yr0, nyr;
  int32_t nmeta;          // staged metas (even, padded): one per X block and window of its row
  int32_t pad[3];
};
static_assert(sizeof(StreamChunkHdr) == 64 && sizeof(StreamBrickHdr) == 16, "headers are fetched with 16-byte loads");

struct StreamPlan {
  bool ok = false;            // false: shapes / sizes outside this format -> caller keeps the gather kernel
  std::string why;
  bool persist = false;
  int nwarps = 0;
  int64_t max_smem = 0;       // dynamic shared memory of the largest brick
  std::vector<StreamBrickHdr> bricks;
  std::vector<StreamChunkHdr> chunks;
  std::vector<StreamRun> xruns, yruns;
  std::vector<StreamEntry> entries;
  std::vector<StreamPass> passes;
  std::vector<StreamMeta> meta;
  std::vector<int32_t> brick_maxrow;   // per brick: the largest X row it reads (direct) / its C row (persist)
  int64_t nbricks() const { return (int64_t)bricks.size(); }
  int64_t nchunks() const { return (int64_t)chunks.size(); }
};

struct StreamShape { int M, K, N; };   // C blocks M x N, X blocks M x K, Y blocks K x N
inline int stream_xs(int M, int K) { return (M * K + 1) & ~1; }   // staged X block stride in doubles (16-byte rows)
int64_t stream_smem_bytes(const StreamShape& sh, int64_t nx, int64_t nmeta, int64_t ny, int64_t nentries, int64_t npasses);

// piece of an X row: blocks [t0, t1) of row `row`
struct StreamPiece { int32_t row, t0, t1; };
struct StreamChunkDef { std::vector<StreamPiece> pieces; };
struct StreamBrickDef {
  std::vector<StreamChunkDef> chunks;
  bool direct = true;
  int32_t s0 = 0, s1 = 0;   // persist bricks: the window [s0, s1) of the C row's slots this brick computes (at most 32)
};

// builds the flat plan of C = X*Y for the given bricks.  pairptr/off_x: per C slot the ordered products (HostPlan).
void stream_build(const StreamShape& sh, int nwarps, int64_t smem_budget, const std::vector<StreamBrickDef>& bricks,
                  const int32_t* rowptr_x, const int32_t* colidx_x, const int32_t* rowptr_y, const int32_t* rowptr_c,
                  const int32_t* pairptr, const uint16_t* off_x, const uint16_t* off_y, StreamPlan& out);

// brick definitions of the two PtAP stages
void stream_bricks_stage1(const HostPlan& hp, const StreamShape& sh, int64_t smem_budget, const int32_t* rowptr_a,
                          const int32_t* colidx_a, const int32_t* rowptr_p, std::vector<StreamBrickDef>& bricks);
void stream_bricks_stage2(const HostPlan& hp, const StreamShape& sh, int nwarps, int64_t smem_budget,
                          const int32_t* rowptr_r, const int32_t* colidx_r, std::vector<StreamBrickDef>& bricks);

}  // namespace bsramg
