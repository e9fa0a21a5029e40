// ptap_prog.h -- "lane programs": the schedule format of the numeric PtAP kernels (host builder: ptap_prog.cpp,
// kernels: ptap_prog.cu).
//
// One block product C = X * Y (stage 1: X = A, Y = P, C = AP; stage 2: X = R, Y = AP, C = A_c) is
// cut into BRICKS, one CTA each.  A brick stages the X blocks of its rows and every Y block they meet in shared memory
// and then runs a PROGRAM: every lane walks its own list of block products (32-bit descriptors: staged X slot, staged
// Y slot, "store" flag), accumulating one output block in registers at a time.  Measured on B200: a shared-memory
// LDS.128 occupies the pipe 4 cycles per warp instruction however few lanes are active, twice that with random bank
// conflicts, and fp64 FMAs overlap it completely (profiles/r2_microbench.md) -- so the schedule keeps all 32 lanes
// busy on every step and makes the loads conflict free by construction:
//   * every output column J of the brick belongs to one of 8 CLASSES; a lane only ever works on columns of the
//     class (lane mod 8), and the staged Y blocks of a class live in slots = class (mod 8): the eight lanes of a
//     quarter warp always read eight different 16-byte bank groups;
//   * the lists of a class are laid end to end and cut into equal shares for the class's lanes, so no lane idles
//     while another still multiplies;
//   * a warp's program is a sequence of ROUNDS of equal length; a lane's list may only end at the end of a round, where
//     the lanes that finished a list park their block in an output-ordered shared staging area with ONE warp-wide
//     store sequence (a store instruction costs the same with 1 or 32 active lanes, and scattered 16-byte global
//     stores cost 12 cycles per block).  Lists longer than a lane's share are cut into parts on several lanes; the
//     extra parts go to overflow slots and are added in a fixed order before the brick's rows leave shared memory
//     with TMA bulk stores (contiguous bs_r*bs_c runs).
// The plan is RELATIVE: a program only holds slots and offsets inside the brick; the matrix rows it applies to come
// from the brick's INSTANCE table.  Bricks with the same relative structure share one program (on a structured mesh
// a handful of programs cover the whole matrix), which is the paper's "coordinates declared once" block COO plan
// in gather form: no index search, no atomics in the hot kernels, fixed summation order.
#pragma once
#include <cstdint>
#include <memory>

#include <cuda_runtime.h>

#include <string>
#include <vector>

namespace bsramg {

constexpr int PROG_NT = 128;             // threads per brick
constexpr int PROG_NW = PROG_NT / 32;    // warps per brick
constexpr int PROG_NCLASS = 8;           // lanes of a quarter warp = column classes
constexpr int PROG_LPC = PROG_NT / PROG_NCLASS;   // lanes per class
constexpr uint32_t PROG_NONE = 0xffffffffu;

struct ProgShape { int M, K, N; };   // C blocks M x N, X blocks M x K, Y blocks K x N

// staged block strides, in doubles (X) and in 16-byte units (Y): blocks are padded to 16 bytes, and Y slots to an
// odd number of 16-byte units so that consecutive slots fall into consecutive bank groups
inline int prog_xs(const ProgShape& s) { return (s.M * s.K + 1) & ~1; }
inline int prog_yc16(const ProgShape& s) { const int c = (s.K * s.N + 1) / 2; return (c & 1) ? c : c + 1; }

struct XRun { uint16_t row, k0, n, dst; };      // X blocks [k0, k0+n) of brick row `row` -> staged slots dst..
struct YCopy { uint16_t yrow, q, slot, pad; };  // block q of staged Y row `yrow` -> Y slot

struct ProgChunk {          // one chunk of a program on the host (offsets into the Program's arrays)
  int32_t xrun0, nxrun;     // XRun range
  int32_t ycopy0, nycopy;   // YCopy range
  int32_t nx, nyslots;      // staged X blocks (8 zero blocks are appended) and Y slots (slots 0..7 are zero blocks)
  int32_t blob0, blob_words;  // the chunk's program words: per warp, per round, wlen descriptor rows of 32 lanes and
                              // (direct mode) one row of store words
  int16_t wrounds[PROG_NW], wlen[PROG_NW];   // rounds of each warp and steps per round
};

// Device format.  rec[]: one RECORD per brick = { blob offset (words), blob words, nrows, nyrows, xsrc[nrows],
// outbase[nrows], ysrc[nyrows] } padded to 16 bytes; rec_off[b] = first word of brick b's record.  blob[]: per program
// and chunk a BLOB = 16 header words (PROG_H_*), the X runs (2 words each: row | k0 << 16, n | dst << 16), the Y copies
// (1 word each: yrow | q << 12 | slot << 20), the program words, and after the last chunk's program words the tables
// crow[nrows] (first staged output block | blocks << 16), fix[2 * nfix] (output slot | first overflow slot << 16, parts)
// and, in persist mode, pstore[PROG_NT].  A persistent CTA fetches the next brick's record while it works on this one,
// then the blob (shared by all bricks of the program, so it comes from L2) and the operands.
enum { PROG_H_NX = 0, PROG_H_NYSLOTS, PROG_H_NXRUN, PROG_H_NYCOPY, PROG_H_ROUNDS01, PROG_H_ROUNDS23, PROG_H_LEN01,
       PROG_H_LEN23, PROG_H_PROG_WORDS, PROG_H_NCS, PROG_H_NOVF, PROG_H_NFIX, PROG_H_NEXT_BLOB, PROG_H_NEXT_WORDS,
       PROG_H_PAD0, PROG_H_PAD1, PROG_H_WORDS };

// relative structure of a brick: what a program is built from (and what bricks are compared by)
struct RelBrick {
  std::vector<int32_t> xlen;   // per brick row: blocks in X's row
  std::vector<int32_t> xcol;   // per X block (rows concatenated): staged Y row it multiplies
  std::vector<int32_t> ylen;   // per staged Y row: blocks
  std::vector<int32_t> ycol;   // per Y block: brick-local output column
  std::vector<int32_t> clen;   // per brick row: blocks in C's row
  std::vector<int32_t> ccol;   // per C block: brick-local output column (ascending inside a row)
  int32_t ncols = 0;           // brick-local output columns
  uint64_t hash() const;
  bool operator==(const RelBrick& o) const {
    return xlen == o.xlen && xcol == o.xcol && ylen == o.ylen && ycol == o.ycol && clen == o.clen && ccol == o.ccol;
  }
};

// one program on the host
struct Program {
  bool ok = false;
  std::string why;
  int32_t nrows = 0, nyrows = 0, nout = 0;
  std::vector<ProgChunk> chunks;     // offsets relative to this program's arrays
  std::vector<XRun> xruns;
  std::vector<YCopy> ycopies;
  std::vector<uint32_t> blob;
  std::vector<uint32_t> tabs;        // crow[nrows], fix[2 * nfix], pstore[PROG_NT] (persist)
  int32_t ncs = 0, novf = 0, nfix = 0;
  int64_t smem = 0;                  // dynamic shared memory the program needs (low + cs of its largest chunk)
  int64_t smem_low = 0, smem_cs = 0;
  int64_t rec_bytes = 0, blob_bytes = 0, xy_bytes = 0;   // one record, the largest blob, the largest X + Y area
  // statistics
  int64_t products = 0, lane_steps = 0, yslots_used = 0;
  int64_t cost = 0;                  // modelled shared-memory cycles of the brick (slowest warp)
};

struct ProgStats {
  int64_t bricks = 0, programs = 0, products = 0, lane_steps = 0, max_smem = 0, plan_bytes = 0;
  int64_t xq_clk = 0, yq_clk = 0;    // modelled shared-memory cycles of the X / Y loads (quarter-warp bank model)
};

// the whole plan of one stage
struct ProgPlan {
  bool ok = false, persist = false;
  std::string why;
  ProgShape shape{0, 0, 0};
  std::vector<int32_t> rec_off;      // nbricks + 1 entries (words)
  std::vector<uint32_t> rec, blob;
  int64_t nbricks = 0, nprograms = 0, nchunks = 0, nycopies = 0;
  int64_t max_smem = 0;              // dynamic shared memory per CTA: records + the largest lower part + the largest staging area
  int32_t rec_max_bytes = 0, blob_max_bytes = 0;
  ProgStats stats;
  std::vector<int64_t> prog_uses;    // bricks per program
  // filled on request (tests): the distinct programs with the relative structures they were built from
  std::vector<std::pair<RelBrick, std::shared_ptr<Program>>> kept;
  std::vector<int32_t> kept_id;      // program id of kept[e] (-1: built but unused)
};

// shared memory of one chunk: `low` = records + blob + X + Y (what is staged per chunk), `cs` = the output staging area
// (kept at the top of the CTA's shared memory so that the next brick can be staged while this one's rows still leave)
struct ProgSmem { int64_t low, cs, rec, blob, xy; int64_t total() const { return low + cs; } };
ProgSmem prog_smem_bytes(const ProgShape& sh, bool persist, bool last_chunk, int32_t nrows, int32_t nyrows, int32_t nfix,
                         int32_t ncs_all, const ProgChunk& ch);
int64_t prog_blob_words(bool persist, bool last_chunk, int32_t nrows, int32_t nfix, const ProgChunk& ch);
inline int32_t prog_rec_words(int32_t nrows, int32_t nyrows) { return (4 + 2 * nrows + nyrows + 3) & ~3; }

// builds the program of one brick.  persist: the brick is ONE row whose inner dimension is cut into chunks that fit
// `budget`; every lane keeps one partial output block over all chunks and the partial blocks of a column are added
// in lane order through shared memory (atomic-free segmented sum).  direct: one chunk, every
// output block is written once from registers.
void prog_build(const ProgShape& sh, bool persist, int64_t budget, int round_len, const RelBrick& rb, Program& out);

// checks a program against the relative structure it was built from: every block product of every output block
// appears exactly once, on a lane of the right class, reading the staged copy of the right blocks.  Integer work only.
bool prog_verify(const ProgShape& sh, bool persist, const RelBrick& rb, const Program& p, std::string& why,
                 ProgStats* stats);

// stage plans.  rows_of_brick: bricks as lists of rows of X (stage 1: fine rows grouped by home aggregate and cut
// to the budget inside; stage 2: one coarse row per brick).
void prog_plan_stage1(const ProgShape& sh, int64_t budget, int round_len, int32_t nrows, const int32_t* rowptr_a,
                      const int32_t* colidx_a, const int32_t* rowptr_p, const int32_t* colidx_p, int32_t ncols_p,
                      const int32_t* rowptr_ap, const int32_t* colidx_ap, ProgPlan& out, bool keep = false);
void prog_plan_stage2(const ProgShape& sh, int64_t budget, int32_t nrows_c, const int32_t* rowptr_r,
                      const int32_t* colidx_r, const int32_t* rowptr_ap, const int32_t* colidx_ap,
                      const int32_t* rowptr_c, const int32_t* colidx_c, ProgPlan& out, bool keep = false);

// ------------------------------------------------------------------ device side
struct ProgArgs {   // all device pointers
  const int32_t* rec_off;
  const uint32_t* rec;
  const uint32_t* blob;
  const double *xvals, *yvals;
  double* cvals;
  int32_t nbricks, rec_max_bytes, blob_max_bytes, smem_total;
};

struct ProgDev {    // device copy of a ProgPlan
  bool ok = false, persist = false;
  ProgShape shape{0, 0, 0};
  int64_t nbricks = 0, nprograms = 0, smem = 0, bytes = 0;
  int32_t grid = 0;                  // persistent CTAs: resident CTAs per SM x SMs (or fewer bricks)
  ProgArgs args{};
  std::vector<void*> owned;
};

int prog_upload(const ProgPlan& pp, ProgDev& pd, cudaStream_t st);
void prog_release(ProgDev& pd);
// prepare = true: cold call that opts the kernel in to the device's dynamic shared memory; false: the hot launch
int prog_launch(const ProgShape& sh, bool persist, const ProgArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st,
                bool prepare, int* ctas_per_sm = nullptr);

// process-wide options of the cold calls (bsr_set_option)
struct Options {
  int64_t force_gather = 0;                 // 1: ptap_symbolic keeps the gather kernels (tests of the fallback)
  int64_t round_len = 0;                    // stage 1: steps between two store points of a warp (0: per program)
  int64_t smem_stage1 = 112 * 1024;         // shared memory a stage-1 brick may use (two bricks per SM)
  int64_t smem_stage2 = 75000;              // stage 2: three coarse rows per SM (register-limited)
};
Options& options();

}  // namespace bsramg
