// ptap_plan.cpp -- host side of ptap_symbolic: structures of AP and A_c and the block coordinate plan.
//
// "the symbolic setup is computed once and reused, while the numeric coarse operators are
// recomputed".  PAPER.md:97-99, 248-250: the blocked COO plan (block coordinates declared once, duplicate-summation
// map built once, every numeric assembly sums contiguous bs_r*bs_c runs).  Here the plan is kept in GATHER form:
// the block products that land on one output block are stored contiguously, in a fixed order (ascending inner
// index), so the numeric kernels sum each output block in registers and write it once -- a segmented sum instead
// of a scatter, hence no atomics and bit-reproducible results.
//
// Structures are symbolic (boolean products; a block is kept even if it is numerically zero) and columns are
// strictly ascending -- the canonical form in which "bit-exact structure" is meaningful (reading R5).
// Cold path: runs on the host cores with OpenMP; nothing here is called by the hot entry points.
#include <algorithm>
#include <cstring>

#include "internal.h"

namespace bsramg {

namespace {

// exclusive prefix sum of per-row counts into a rowptr-like array; returns the total (as int64)
int64_t prefix(const std::vector<int32_t>& cnt, std::vector<int32_t>& ptr) {
  ptr.resize(cnt.size() + 1);
  int64_t s = 0;
  for (size_t i = 0; i < cnt.size(); ++i) {
    ptr[i] = (int32_t)s;
    s += cnt[i];
  }
  ptr[cnt.size()] = (int32_t)s;
  return s;
}

// One product C = X * Y of two block-sparse patterns, output-stationary:
//   for row i of X: every (x-slot a in row i, y-slot b in row col_x[a]) is one block product landing on column
//   col_y[b].  Products are grouped by output column (ascending) and ordered by ascending a inside a group.
// Emits the structure of C (rowptr/colidx/rowidx), per-output-slot product ranges (pairptr) and per product the
// offsets (a - rowptr_x[i], b - rowptr_y[col_x[a]]).
struct Product {
  std::vector<int32_t>*rowptr_c, *colidx_c, *rowidx_c, *pairptr;
  std::vector<uint16_t>*off_x, *off_y;
  int32_t max_off_x = 0, max_off_y = 0;
};

int symbolic_product(int32_t nrows, const int32_t* rowptr_x, const int32_t* colidx_x, const int32_t* rowptr_y,
                     const int32_t* colidx_y, Product& out, std::string& err) {
  std::vector<int32_t> nblk((size_t)nrows), nprod((size_t)nrows);
  int bad = 0;
  // pass 1: counts per row
#pragma omp parallel
  {
    std::vector<uint64_t> keys;
#pragma omp for schedule(dynamic, 256) reduction(| : bad)
    for (int32_t i = 0; i < nrows; ++i) {
      keys.clear();
      for (int32_t a = rowptr_x[i]; a < rowptr_x[i + 1]; ++a) {
        const int32_t j = colidx_x[a];
        if (a - rowptr_x[i] > 0xffff || rowptr_y[j + 1] - rowptr_y[j] > 0x10000) bad |= 1;
        for (int32_t b = rowptr_y[j]; b < rowptr_y[j + 1]; ++b) keys.push_back((uint64_t)(uint32_t)colidx_y[b]);
      }
      std::sort(keys.begin(), keys.end());
      nprod[i] = (int32_t)keys.size();
      nblk[i] = (int32_t)(std::unique(keys.begin(), keys.end()) - keys.begin());
    }
  }
  if (bad) { err = "row longer than 65536 blocks"; return BSR_ERR_LIMIT; }
  std::vector<int32_t> prodptr;
  const int64_t nc = prefix(nblk, *out.rowptr_c);
  const int64_t np = prefix(nprod, prodptr);
  if (nc >= (1LL << 31) || np >= (1LL << 31)) { err = "more than 2^31 blocks or block products"; return BSR_ERR_LIMIT; }
  out.colidx_c->resize((size_t)nc);
  out.rowidx_c->resize((size_t)nc);
  out.pairptr->resize((size_t)nc + 1);
  out.off_x->resize((size_t)np);
  out.off_y->resize((size_t)np);
  (*out.pairptr)[(size_t)nc] = (int32_t)np;
  int32_t mx = 0, my = 0;
  // pass 2: fill.  key = (output column, offset in X's row, offset in Y's row); sorting groups by column and
  // orders each group by ascending x-slot, i.e. ascending inner index.
#pragma omp parallel
  {
    std::vector<uint64_t> keys;
#pragma omp for schedule(dynamic, 256) reduction(max : mx) reduction(max : my)
    for (int32_t i = 0; i < nrows; ++i) {
      keys.clear();
      for (int32_t a = rowptr_x[i]; a < rowptr_x[i + 1]; ++a) {
        const int32_t j = colidx_x[a];
        const uint64_t oa = (uint64_t)(a - rowptr_x[i]);
        for (int32_t b = rowptr_y[j]; b < rowptr_y[j + 1]; ++b)
          keys.push_back(((uint64_t)(uint32_t)colidx_y[b] << 32) | (oa << 16) | (uint64_t)(b - rowptr_y[j]));
      }
      std::sort(keys.begin(), keys.end());
      int32_t slot = (*out.rowptr_c)[i] - 1;
      int32_t p = prodptr[i];
      int64_t last = -1;
      for (uint64_t key : keys) {
        const int64_t col = (int64_t)(key >> 32);
        if (col != last) {
          ++slot;
          (*out.colidx_c)[slot] = (int32_t)col;
          (*out.rowidx_c)[slot] = i;
          (*out.pairptr)[slot] = p;
          last = col;
        }
        const int32_t ox = (int32_t)((key >> 16) & 0xffff), oy = (int32_t)(key & 0xffff);
        (*out.off_x)[p] = (uint16_t)ox;
        (*out.off_y)[p] = (uint16_t)oy;
        mx = std::max(mx, ox);
        my = std::max(my, oy);
        ++p;
      }
    }
  }
  out.max_off_x = mx;
  out.max_off_y = my;
  return BSR_OK;
}

}  // namespace

int HostPlan::build_stage1(int32_t nbrows_a_, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p_,
                           const int32_t* rowptr_p, const int32_t* colidx_p) {
  nbrows_a = nbrows_a_;
  nbcols_p = nbcols_p_;
  // stage 1: AP = A * P
  Product s1;
  s1.rowptr_c = &rowptr_ap; s1.colidx_c = &colidx_ap; s1.rowidx_c = &rowidx_ap; s1.pairptr = &pairptr1;
  s1.off_x = &k1; s1.off_y = &q1;
  int rc = symbolic_product(nbrows_a, rowptr_a, colidx_a, rowptr_p, colidx_p, s1, err);
  if (rc != BSR_OK) return rc;
  max_k1 = s1.max_off_x; max_q1 = s1.max_off_y;
  const int64_t nnzb_a = rowptr_a[nbrows_a];
  pstart.resize((size_t)nnzb_a);
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < nnzb_a; ++k) pstart[(size_t)k] = rowptr_p[colidx_a[k]];
  return BSR_OK;
}

int HostPlan::build(int32_t nbrows_a_, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p_,
                    const int32_t* rowptr_p, const int32_t* colidx_p, const int32_t* rowptr_r,
                    const int32_t* colidx_r) {
  int rc = build_stage1(nbrows_a_, rowptr_a, colidx_a, nbcols_p_, rowptr_p, colidx_p);
  if (rc != BSR_OK) return rc;
  // stage 2: A_c = R * AP
  Product st2;
  st2.rowptr_c = &rowptr_c; st2.colidx_c = &colidx_c; st2.rowidx_c = &rowidx_c; st2.pairptr = &pairptr2;
  st2.off_x = &t2; st2.off_y = &s2;
  rc = symbolic_product(nbcols_p, rowptr_r, colidx_r, rowptr_ap.data(), colidx_ap.data(), st2, err);
  if (rc != BSR_OK) return rc;
  max_t2 = st2.max_off_x; max_s2 = st2.max_off_y;
  // row starts of the gathered operand, one per slot of the left operand (saves one indirection in the kernels)
  const int64_t nnzb_r = rowptr_r[nbcols_p];
  apstart.resize((size_t)nnzb_r);
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < nnzb_r; ++t) apstart[(size_t)t] = rowptr_ap[(size_t)colidx_r[t]];
  return BSR_OK;
}

// ------------------------------------------------------------------ C ABI for CPU-side tests of the plan
}  // namespace bsramg

using namespace bsramg;

extern "C" {

struct ptap_host_plan_s {
  HostPlan plan;
  std::vector<int32_t> rowptr_r, colidx_r, perm_r;
  std::vector<int32_t> rowptr_a, colidx_a, rowptr_p;   // copies, for ptap_host_stream_stats
};

void* ptap_host_plan_build(int32_t nbrows_a, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p,
                           const int32_t* rowptr_p, const int32_t* colidx_p) {
  if (!rowptr_a || !colidx_a || !rowptr_p || !colidx_p || nbrows_a < 0 || nbcols_p < 0) {
    fail(BSR_ERR_NULL, "ptap_host_plan_build: bad argument");
    return nullptr;
  }
  ptap_host_plan_s* h = new (std::nothrow) ptap_host_plan_s();
  if (!h) { fail(BSR_ERR_ALLOC, "host allocation failed"); return nullptr; }
  host_transpose_structure(nbrows_a, nbcols_p, rowptr_p, colidx_p, h->rowptr_r, h->colidx_r, h->perm_r);
  h->rowptr_a.assign(rowptr_a, rowptr_a + nbrows_a + 1);
  h->colidx_a.assign(colidx_a, colidx_a + rowptr_a[nbrows_a]);
  h->rowptr_p.assign(rowptr_p, rowptr_p + nbrows_a + 1);
  int rc = h->plan.build(nbrows_a, rowptr_a, colidx_a, nbcols_p, rowptr_p, colidx_p, h->rowptr_r.data(),
                         h->colidx_r.data());
  if (rc != BSR_OK) {
    fail(rc, "%s", h->plan.err.c_str());
    delete h;
    return nullptr;
  }
  return h;
}

int ptap_host_plan_get(void* handle, const char* name, const void** ptr, int64_t* count, int32_t* elem_bytes) {
  if (!handle || !name || !ptr || !count || !elem_bytes) return fail(BSR_ERR_NULL, "ptap_host_plan_get: null argument");
  ptap_host_plan_s* h = (ptap_host_plan_s*)handle;
  HostPlan& p = h->plan;
#define I32(field, vec) if (!strcmp(name, field)) { *ptr = (vec).data(); *count = (int64_t)(vec).size(); *elem_bytes = 4; return BSR_OK; }
#define U16(field, vec) if (!strcmp(name, field)) { *ptr = (vec).data(); *count = (int64_t)(vec).size(); *elem_bytes = 2; return BSR_OK; }
  I32("rowptr_ap", p.rowptr_ap) I32("colidx_ap", p.colidx_ap) I32("rowidx_ap", p.rowidx_ap)
  I32("rowptr_c", p.rowptr_c) I32("colidx_c", p.colidx_c) I32("rowidx_c", p.rowidx_c)
  I32("pairptr1", p.pairptr1) U16("k1", p.k1) U16("q1", p.q1) I32("pstart", p.pstart)
  I32("pairptr2", p.pairptr2) U16("t2", p.t2) U16("s2", p.s2) I32("apstart", p.apstart)
  I32("rowptr_r", h->rowptr_r) I32("colidx_r", h->colidx_r) I32("perm_r", h->perm_r)
#undef I32
#undef U16
  return fail(BSR_ERR_NULL, "ptap_host_plan_get: unknown array '%s'", name);
}

int ptap_host_stream_stats(void* handle, int32_t bs_f, int32_t bs_c, int32_t stage, int64_t smem_budget,
                           int64_t* out8) {
  if (!handle || !out8 || (stage != 1 && stage != 2)) return fail(BSR_ERR_NULL, "ptap_host_stream_stats: bad argument");
  ptap_host_plan_s* h = (ptap_host_plan_s*)handle;
  const HostPlan& hp = h->plan;
  std::vector<StreamBrickDef> bricks;
  StreamPlan sp;
  if (stage == 1) {
    const StreamShape sh{bs_f, bs_f, bs_c};
    stream_bricks_stage1(hp, sh, smem_budget, h->rowptr_a.data(), h->colidx_a.data(), h->rowptr_p.data(), bricks);
    stream_build(sh, 8, smem_budget, bricks, h->rowptr_a.data(), h->colidx_a.data(), h->rowptr_p.data(),
                 hp.rowptr_ap.data(), hp.pairptr1.data(), hp.k1.data(), hp.q1.data(), sp);
  } else {
    const StreamShape sh{bs_c, bs_f, bs_c};
    stream_bricks_stage2(hp, sh, 4, smem_budget, h->rowptr_r.data(), h->colidx_r.data(), bricks);
    stream_build(sh, 4, smem_budget, bricks, h->rowptr_r.data(), h->colidx_r.data(), hp.rowptr_ap.data(),
                 hp.rowptr_c.data(), hp.pairptr2.data(), hp.t2.data(), hp.s2.data(), sp);
  }
  int64_t bits = 0, lanes = 0, steps = 0;
  for (const StreamMeta& m : sp.meta) bits += __builtin_popcount(m.mask);
  for (const StreamEntry& e : sp.entries) lanes += e.nslots();
  for (const StreamPass& p : sp.passes) steps += p.steps;
  out8[0] = sp.ok ? 1 : 0; out8[1] = sp.nbricks(); out8[2] = sp.nchunks(); out8[3] = sp.max_smem;
  out8[4] = bits; out8[5] = lanes; out8[6] = (int64_t)sp.passes.size(); out8[7] = steps;
  return BSR_OK;
}

void ptap_host_plan_free(void* handle) { delete (ptap_host_plan_s*)handle; }

}  // extern "C"

namespace bsramg {

}  // namespace bsramg
