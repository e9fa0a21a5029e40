// ptap_stream.cpp -- host side (cold) of the brick-staged numeric PtAP: cuts the two block products of ptap_numeric
// into bricks, chunks and items (internal.h, "brick-staged product streams").
//
// the blocked COO plan is built once ("coordinates declared once ... duplicate-summation
// map") and every numeric assembly reuses it.  Here that map is a schedule: which CTA stages which blocks of the two
// operands in shared memory, which lane group sums which run of products, and in which fixed order partial blocks
// are added into the coarse block they belong to -- so the hot kernels do no index search and use no atomics.
// stage 1 is the dominant fine-level product AP = A*P (<3,3,6>), stage 2 the R*(AP) product.
//
// Integer work only; OpenMP over bricks; nothing here runs in the hot calls.
#include <algorithm>
#include <climits>
#include <cstring>
#include <numeric>
#include <queue>

#include "internal.h"

namespace bsramg {

static inline int64_t up16(int64_t b) { return (b + 15) & ~int64_t(15); }

int64_t stream_smem_bytes(const StreamShape& sh, int64_t nx, int64_t nmeta, int64_t ny, int64_t nentries, int64_t npasses) {
  int64_t b = 0;
  b += up16(nx * stream_xs(sh.M, sh.K) * 8);
  b += up16(nmeta * (int64_t)sizeof(StreamMeta));
  b += up16(ny * sh.K * sh.N * 8);
  b += up16(nentries * (int64_t)sizeof(StreamEntry));
  b += up16(npasses * (int64_t)sizeof(StreamPass));
  return b;
}

namespace {

struct LocalChunk {
  std::vector<StreamRun> xruns, yruns;
  std::vector<StreamEntry> entries;
  std::vector<StreamPass> passes;
  std::vector<StreamMeta> meta;
  int32_t nx = 0, ny = 0;
};
struct LocalBrick {
  std::vector<LocalChunk> chunks;
  int32_t out = 0, nslots = 0;
  bool bad = false;
};

inline int popc32(uint32_t v) { return __builtin_popcount(v); }

}  // namespace

void stream_build(const StreamShape& sh, int nwarps, int64_t smem_budget, const std::vector<StreamBrickDef>& bricks,
                  const int32_t* rowptr_x, const int32_t* colidx_x, const int32_t* rowptr_y, const int32_t* rowptr_c,
                  const int32_t* pairptr, const uint16_t* off_x, const uint16_t* off_y, StreamPlan& out) {
  out = StreamPlan();
  out.nwarps = nwarps;
  const int64_t nb = (int64_t)bricks.size();
  out.persist = nb > 0 && !bricks[0].direct;
  std::vector<LocalBrick> L((size_t)nb);

#pragma omp parallel
  {
    std::vector<int32_t> ycols, ydst, order, first, last;
#pragma omp for schedule(dynamic, 16)
    for (int64_t b = 0; b < nb; ++b) {
      const StreamBrickDef& bd = bricks[(size_t)b];
      LocalBrick& lb = L[(size_t)b];
      if (bd.direct == out.persist) { lb.bad = true; continue; }  // one mode per plan
      int32_t prow = -1;
      if (!bd.direct) {
        // persist: one window of one C row per brick, one piece per chunk
        for (const auto& cd : bd.chunks) {
          if (cd.pieces.size() != 1 || (prow >= 0 && cd.pieces[0].row != prow)) lb.bad = true;
          if (!cd.pieces.empty()) prow = cd.pieces[0].row;
        }
        if (prow < 0) { lb.bad = true; continue; }
        const int32_t ns = rowptr_c[prow + 1] - rowptr_c[prow];
        if (bd.s0 < 0 || bd.s1 > ns || bd.s1 - bd.s0 > 32 || (bd.s1 <= bd.s0 && ns > 0)) { lb.bad = true; continue; }
        lb.out = rowptr_c[prow] + bd.s0;
        lb.nslots = bd.s1 - bd.s0;
      }
      if (lb.bad) continue;
      lb.chunks.resize(bd.chunks.size());
      for (size_t ci = 0; ci < bd.chunks.size(); ++ci) {
        const StreamChunkDef& cd = bd.chunks[ci];
        LocalChunk& lc = lb.chunks[ci];
        // ---- X runs
        std::vector<int32_t> piece_xbase(cd.pieces.size()), piece_mbase(cd.pieces.size()), piece_nwin(cd.pieces.size());
        ycols.clear();
        int32_t dst = 0, nmeta = 0;
        for (size_t pi = 0; pi < cd.pieces.size(); ++pi) {
          const StreamPiece& pc = cd.pieces[pi];
          const int32_t src = rowptr_x[pc.row] + pc.t0, n = pc.t1 - pc.t0;
          const int32_t ns = rowptr_c[pc.row + 1] - rowptr_c[pc.row];
          piece_xbase[pi] = dst;
          piece_mbase[pi] = nmeta;
          piece_nwin[pi] = bd.direct ? std::max(1, (ns + 31) / 32) : 1;
          if (n > 0xffff) lb.bad = true;
          if (n <= 0) continue;
          if (!lc.xruns.empty() && lc.xruns.back().src + lc.xruns.back().n == src) lc.xruns.back().n += n;
          else lc.xruns.push_back({src, n, dst});
          if (bd.direct)
            for (int32_t k = src; k < src + n; ++k) ycols.push_back(colidx_x[k]);
          dst += n;
          nmeta += n * piece_nwin[pi];
        }
        if (lb.bad) break;
        // ---- masks per (X block, window) and the products' Y block range per (X block, window)
        lc.meta.assign((size_t)nmeta, StreamMeta{0u, 0u});
        first.assign((size_t)nmeta, INT32_MAX);
        last.assign((size_t)nmeta, -1);
        for (size_t pi = 0; pi < cd.pieces.size(); ++pi) {
          const StreamPiece& pc = cd.pieces[pi];
          const int32_t len = pc.t1 - pc.t0;
          const int32_t r0 = rowptr_c[pc.row], ns = rowptr_c[pc.row + 1] - r0;
          const int32_t sa = bd.direct ? 0 : bd.s0, sb = bd.direct ? ns : bd.s1;
          for (int32_t sl = sa; sl < sb; ++sl) {
            const int32_t w = bd.direct ? sl / 32 : 0, bit = bd.direct ? sl % 32 : sl - bd.s0;
            for (int64_t p = pairptr[r0 + sl]; p < pairptr[r0 + sl + 1]; ++p) {
              const int32_t ox = off_x[p];
              if (ox < pc.t0 || ox >= pc.t1) continue;
              const size_t m = (size_t)piece_mbase[pi] + (size_t)w * len + (ox - pc.t0);
              lc.meta[m].mask |= 1u << bit;
              first[m] = std::min(first[m], (int32_t)off_y[p]);
              last[m] = std::max(last[m], (int32_t)off_y[p]);
            }
          }
        }
        // ---- Y runs.  Direct: every referenced Y row once, whole.  Persist: per X block the blocks of its Y row
        // that fall into the brick's window (a contiguous piece of the row: its columns ascend with the slots).
        int32_t yd = 0;
        if (bd.direct) {
          std::sort(ycols.begin(), ycols.end());
          ycols.erase(std::unique(ycols.begin(), ycols.end()), ycols.end());
          ydst.resize(ycols.size());
          for (size_t t = 0; t < ycols.size(); ++t) {
            const int32_t j = ycols[t], src = rowptr_y[j], n = rowptr_y[j + 1] - rowptr_y[j];
            ydst[t] = yd;
            if (n > 0) {
              if (!lc.yruns.empty() && lc.yruns.back().src + lc.yruns.back().n == src) lc.yruns.back().n += n;
              else lc.yruns.push_back({src, n, yd});
            }
            yd += n;
          }
          for (size_t pi = 0; pi < cd.pieces.size(); ++pi) {
            const StreamPiece& pc = cd.pieces[pi];
            const int32_t len = pc.t1 - pc.t0;
            for (int32_t w = 0; w < piece_nwin[pi]; ++w)
              for (int32_t k = 0; k < len; ++k) {
                const size_t m = (size_t)piece_mbase[pi] + (size_t)w * len + k;
                if (!lc.meta[m].mask) continue;
                const int32_t j = colidx_x[rowptr_x[pc.row] + pc.t0 + k];
                lc.meta[m].ybase = (uint32_t)(ydst[(size_t)(std::lower_bound(ycols.begin(), ycols.end(), j) - ycols.begin())] + first[m]);
              }
          }
        } else {
          const StreamPiece& pc = cd.pieces[0];
          for (int32_t k = 0; k < pc.t1 - pc.t0; ++k) {
            const size_t m = (size_t)piece_mbase[0] + k;
            if (!lc.meta[m].mask) continue;
            const int32_t j = colidx_x[rowptr_x[pc.row] + pc.t0 + k];
            const int32_t src = rowptr_y[j] + first[m], n = last[m] - first[m] + 1;
            lc.meta[m].ybase = (uint32_t)yd;
            if (!lc.yruns.empty() && lc.yruns.back().src + lc.yruns.back().n == src && lc.yruns.back().dst + lc.yruns.back().n == yd)
              lc.yruns.back().n += n;
            else lc.yruns.push_back({src, n, yd});
            yd += n;
          }
        }
        lc.ny = yd;
        // the lane of a slot reads block rank(slot) of the window's piece of the Y row: must be the product's own block
        for (size_t pi = 0; pi < cd.pieces.size() && !lb.bad; ++pi) {
          const StreamPiece& pc = cd.pieces[pi];
          const int32_t len = pc.t1 - pc.t0;
          const int32_t r0 = rowptr_c[pc.row], ns = rowptr_c[pc.row + 1] - r0;
          const int32_t sa = bd.direct ? 0 : bd.s0, sb = bd.direct ? ns : bd.s1;
          for (int32_t sl = sa; sl < sb && !lb.bad; ++sl) {
            const int32_t w = bd.direct ? sl / 32 : 0, bit = bd.direct ? sl % 32 : sl - bd.s0;
            for (int64_t p = pairptr[r0 + sl]; p < pairptr[r0 + sl + 1]; ++p) {
              const int32_t ox = off_x[p];
              if (ox < pc.t0 || ox >= pc.t1) continue;
              const size_t m = (size_t)piece_mbase[pi] + (size_t)w * len + (ox - pc.t0);
              if (popc32(lc.meta[m].mask & ((1u << bit) - 1u)) + first[m] != (int)off_y[p]) { lb.bad = true; break; }
            }
          }
        }
        if (lb.bad) break;
        lc.nx = dst;
        if (lc.meta.size() & 1) lc.meta.push_back(StreamMeta{0u, 0u});  // even count: 16-byte staging
        // ---- passes
        if (bd.direct) {
          // the output blocks of all rows, longest rows first, laid end to end and cut every 32 lanes and at every
          // window boundary: a pass holds whole (windows of) rows and at most two fragments
          const size_t np = cd.pieces.size();
          order.resize(np);
          std::iota(order.begin(), order.end(), 0);
          auto nsl = [&](int32_t pi) { return rowptr_c[cd.pieces[(size_t)pi].row + 1] - rowptr_c[cd.pieces[(size_t)pi].row]; };
          auto plen = [&](int32_t pi) { return cd.pieces[(size_t)pi].t1 - cd.pieces[(size_t)pi].t0; };
          std::stable_sort(order.begin(), order.end(), [&](int32_t u, int32_t v) { return plen(u) > plen(v); });
          StreamPass ps{0, 0, 0, 0};
          int32_t lane0 = 0;
          auto close_pass = [&]() {
            if ((int32_t)lc.entries.size() > ps.e0) {
              ps.e1 = (int32_t)lc.entries.size();
              lc.passes.push_back(ps);
            }
            ps = StreamPass{(int32_t)lc.entries.size(), 0, 0, 0};
            lane0 = 0;
          };
          for (int32_t pi : order) {
            const StreamPiece& pc = cd.pieces[(size_t)pi];
            if (pc.t0 != 0) lb.bad = true;
            int32_t s0 = 0;
            const int32_t ns = nsl(pi), len = plen(pi);
            while (s0 < ns) {
              const int32_t w = s0 / 32;
              const int32_t take = std::min(std::min(ns - s0, 32 - lane0), 32 * (w + 1) - s0);
              lc.entries.push_back(StreamEntry{rowptr_c[pc.row] + 32 * w, piece_xbase[(size_t)pi],
                                               piece_mbase[(size_t)pi] + w * len, StreamEntry::pack(len, lane0, take, s0 - 32 * w)});
              ps.steps = std::max(ps.steps, len);
              lane0 += take;
              s0 += take;
              if (lane0 == 32) close_pass();
            }
          }
          close_pass();
        } else if (lb.nslots > 0) {
          // the chunk's piece of the row, cut into nwarps contiguous shares: pass w belongs to warp w
          const StreamPiece& pc = cd.pieces[0];
          const int32_t len = pc.t1 - pc.t0;
          for (int w = 0; w < nwarps; ++w) {
            const int32_t a = (int32_t)((int64_t)len * w / nwarps), e = (int32_t)((int64_t)len * (w + 1) / nwarps);
            lc.passes.push_back(StreamPass{(int32_t)lc.entries.size(), (int32_t)lc.entries.size() + 1, e - a, 0});
            lc.entries.push_back(StreamEntry{0, piece_xbase[0] + a, piece_mbase[0] + a, StreamEntry::pack(e - a, 0, lb.nslots, 0)});
          }
        }
      }
    }
  }
  for (const auto& lb : L)
    if (lb.bad) { out.why = "brick outside the staged format (unsorted operand or a row piece longer than 65535 blocks)"; return; }
  // ---- flatten
  int64_t nchunks = 0;
  for (const auto& lb : L) nchunks += (int64_t)lb.chunks.size();
  out.bricks.resize((size_t)nb);
  out.chunks.resize((size_t)nchunks);
  out.brick_maxrow.assign((size_t)nb, 0);
  for (int64_t b = 0; b < nb; ++b)
    for (const auto& cd : bricks[(size_t)b].chunks)
      for (const auto& pc : cd.pieces) out.brick_maxrow[(size_t)b] = std::max(out.brick_maxrow[(size_t)b], pc.row);
  int64_t c = 0, nxr = 0, nyr = 0, nen = 0, npa = 0, nme = 0;
  for (int64_t b = 0; b < nb; ++b) {
    const LocalBrick& lb = L[(size_t)b];
    out.bricks[(size_t)b] = StreamBrickHdr{(int32_t)c, (int32_t)lb.chunks.size(), lb.out, lb.nslots};
    if (out.persist)
      out.max_smem = std::max<int64_t>(out.max_smem, up16((int64_t)nwarps * lb.nslots * sh.M * sh.N * 8));
    for (const auto& lc : lb.chunks) {
      StreamChunkHdr h;
      memset(&h, 0, sizeof h);
      h.meta0 = nme; h.nx = lc.nx; h.ny = lc.ny; h.nmeta = (int32_t)lc.meta.size();
      h.ent0 = (int32_t)nen; h.nent = (int32_t)lc.entries.size();
      h.pass0 = (int32_t)npa; h.npass = (int32_t)lc.passes.size();
      h.xr0 = (int32_t)nxr; h.nxr = (int32_t)lc.xruns.size();
      h.yr0 = (int32_t)nyr; h.nyr = (int32_t)lc.yruns.size();
      out.chunks[(size_t)c] = h;
      out.max_smem = std::max(out.max_smem, stream_smem_bytes(sh, lc.nx, (int64_t)lc.meta.size(), lc.ny,
                                                              (int64_t)lc.entries.size(), (int64_t)lc.passes.size()));
      nxr += (int64_t)lc.xruns.size(); nyr += (int64_t)lc.yruns.size(); nen += (int64_t)lc.entries.size();
      npa += (int64_t)lc.passes.size(); nme += (int64_t)lc.meta.size();  // even per chunk: 16-byte aligned
      ++c;
    }
  }
  if (nen >= (1LL << 31) || nxr >= (1LL << 31) || nyr >= (1LL << 31) || out.max_smem > smem_budget) {
    out.why = out.max_smem > smem_budget ? "a brick does not fit the shared memory budget" : "too many entries";
    return;
  }
  out.xruns.resize((size_t)nxr); out.yruns.resize((size_t)nyr); out.entries.resize((size_t)nen);
  out.passes.resize((size_t)npa); out.meta.assign((size_t)nme, StreamMeta{0u, 0u});
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t b = 0; b < nb; ++b) {
    const LocalBrick& lb = L[(size_t)b];
    int64_t cc = out.bricks[(size_t)b].chunk0;
    for (const auto& lc : lb.chunks) {
      const StreamChunkHdr& h = out.chunks[(size_t)cc];
      std::copy(lc.xruns.begin(), lc.xruns.end(), out.xruns.begin() + h.xr0);
      std::copy(lc.yruns.begin(), lc.yruns.end(), out.yruns.begin() + h.yr0);
      std::copy(lc.entries.begin(), lc.entries.end(), out.entries.begin() + h.ent0);
      std::copy(lc.passes.begin(), lc.passes.end(), out.passes.begin() + h.pass0);
      std::copy(lc.meta.begin(), lc.meta.end(), out.meta.begin() + h.meta0);
      ++cc;
    }
  }
  out.ok = true;
}

// ------------------------------------------------------------------ stage 1 bricks: AP = A*P
// Fine rows that share a "home" coarse column are staged together: home(i) = the column J of AP's row i that
// receives the most products, i.e. argmax_J |N(i) ∩ supp P(:,J)| -- for an aggregation-based P that is i's own
// aggregate, and the P rows the brick references are the aggregate's neighbourhood.  Purely structural; it only
// decides scheduling.  A group that does not fit the shared-memory budget is halved (by row order) until it does.
void stream_bricks_stage1(const HostPlan& hp, const StreamShape& sh, int64_t smem_budget, const int32_t* rowptr_a,
                          const int32_t* colidx_a, const int32_t* rowptr_p, std::vector<StreamBrickDef>& bricks) {
  const int32_t n = hp.nbrows_a, nc = hp.nbcols_p;
  std::vector<int32_t> home((size_t)n, 0);
#pragma omp parallel for schedule(static)
  for (int32_t i = 0; i < n; ++i) {
    int32_t best = -1, bestn = -1;
    for (int32_t s = hp.rowptr_ap[i]; s < hp.rowptr_ap[i + 1]; ++s) {
      const int32_t np = hp.pairptr1[(size_t)s + 1] - hp.pairptr1[s];
      if (np > bestn) { bestn = np; best = hp.colidx_ap[s]; }
    }
    home[i] = best < 0 ? 0 : best;
  }
  // counting sort of the rows by home (stable: ascending row id inside a group)
  std::vector<int32_t> gptr((size_t)nc + 2, 0), grows((size_t)n);
  for (int32_t i = 0; i < n; ++i) gptr[(size_t)home[i] + 1]++;
  for (int32_t j = 0; j < nc; ++j) gptr[(size_t)j + 1] += gptr[j];
  {
    std::vector<int32_t> fill(gptr.begin(), gptr.end() - 1);
    for (int32_t i = 0; i < n; ++i) grows[(size_t)fill[home[i]]++] = i;
  }
  std::vector<std::vector<StreamBrickDef>> per((size_t)nc);
#pragma omp parallel
  {
    std::vector<int32_t> cols;
    std::vector<std::pair<int32_t, int32_t>> stack;
#pragma omp for schedule(dynamic, 64)
    for (int32_t J = 0; J < nc; ++J) {
      stack.clear();
      if (gptr[(size_t)J + 1] > gptr[J]) stack.push_back({gptr[J], gptr[(size_t)J + 1]});
      while (!stack.empty()) {
        const auto r = stack.back();
        stack.pop_back();
        int64_t nx = 0, ny = 0, nmeta = 0, nent = 0, nslot = 0;
        cols.clear();
        for (int32_t t = r.first; t < r.second; ++t) {
          const int32_t i = grows[t];
          const int64_t len = rowptr_a[i + 1] - rowptr_a[i], ns = hp.rowptr_ap[i + 1] - hp.rowptr_ap[i];
          const int64_t nwin = std::max<int64_t>(1, (ns + 31) / 32);   // rows beyond 32 output blocks: one mask set per window
          nx += len; nmeta += len * nwin; nent += nwin + 1; nslot += ns;
          cols.insert(cols.end(), colidx_a + rowptr_a[i], colidx_a + rowptr_a[i + 1]);
        }
        std::sort(cols.begin(), cols.end());
        cols.erase(std::unique(cols.begin(), cols.end()), cols.end());
        for (int32_t j : cols) ny += rowptr_p[j + 1] - rowptr_p[j];
        const int64_t bytes = stream_smem_bytes(sh, nx, nmeta + 1, ny, nent, nslot / 32 + 2);
        if (bytes > smem_budget - 512 && r.second - r.first > 1) {
          const int32_t mid = r.first + (r.second - r.first) / 2;
          stack.push_back({mid, r.second});   // popped after the first half: keeps row order
          stack.push_back({r.first, mid});
          continue;
        }
        StreamBrickDef bd;
        bd.direct = true;
        bd.chunks.resize(1);
        for (int32_t t = r.first; t < r.second; ++t) {
          const int32_t i = grows[t];
          bd.chunks[0].pieces.push_back({i, 0, rowptr_a[i + 1] - rowptr_a[i]});
        }
        per[(size_t)J].push_back(std::move(bd));
      }
    }
  }
  bricks.clear();
  for (auto& v : per)
    for (auto& bd : v) bricks.push_back(std::move(bd));
}

// ------------------------------------------------------------------ stage 2 bricks: A_c = R*(AP)
// One brick per coarse row I.  Its R row is cut into chunks of consecutive blocks such that the chunk's R blocks, the
// AP rows they reference, the codes, items and parts fit the budget next to the row's accumulator.
void stream_bricks_stage2(const HostPlan& hp, const StreamShape& sh, int nwarps, int64_t smem_budget,
                          const int32_t* rowptr_r, const int32_t* colidx_r, std::vector<StreamBrickDef>& bricks) {
  const int32_t nc = hp.nbcols_p;
  // one brick per WINDOW of 32 consecutive slots of a coarse row (one window for the 27-point box stencil)
  std::vector<int64_t> bptr((size_t)nc + 1, 0);
  for (int32_t I = 0; I < nc; ++I) {
    const int32_t ns = hp.rowptr_c[I + 1] - hp.rowptr_c[I];
    bptr[(size_t)I + 1] = bptr[(size_t)I] + std::max(1, (ns + 31) / 32);
  }
  bricks.assign((size_t)bptr[(size_t)nc], StreamBrickDef());
#pragma omp parallel
  {
    std::vector<int32_t> lo, hi;
#pragma omp for schedule(dynamic, 64)
    for (int32_t I = 0; I < nc; ++I) {
      const int32_t len = rowptr_r[I + 1] - rowptr_r[I];
      const int32_t c0 = hp.rowptr_c[I], ns = hp.rowptr_c[I + 1] - c0;
      for (int64_t wb = bptr[(size_t)I]; wb < bptr[(size_t)I + 1]; ++wb) {
        StreamBrickDef& bd = bricks[(size_t)wb];
        bd.direct = false;
        bd.s0 = (int32_t)(wb - bptr[(size_t)I]) * 32;
        bd.s1 = std::min(ns, bd.s0 + 32);
        // blocks of AP's row i that land in this window, per R block t
        lo.assign((size_t)len, INT32_MAX);
        hi.assign((size_t)len, -1);
        for (int32_t sl = bd.s0; sl < bd.s1; ++sl)
          for (int64_t p = hp.pairptr2[(size_t)c0 + sl]; p < hp.pairptr2[(size_t)c0 + sl + 1]; ++p) {
            const int32_t t = hp.t2[(size_t)p], y = hp.s2[(size_t)p];
            lo[(size_t)t] = std::min(lo[(size_t)t], y);
            hi[(size_t)t] = std::max(hi[(size_t)t], y);
          }
        int32_t t0 = 0;
        int64_t nx = 0, ny = 0;
        for (int32_t t = 0; t < len; ++t) {
          const int64_t ay = hi[(size_t)t] >= 0 ? hi[(size_t)t] - lo[(size_t)t] + 1 : 0;
          if (stream_smem_bytes(sh, nx + 1, nx + 2, ny + ay, nwarps, nwarps) > smem_budget - 512 && t > t0) {
            bd.chunks.push_back(StreamChunkDef{{StreamPiece{I, t0, t}}});
            t0 = t; nx = 0; ny = 0;
          }
          nx += 1; ny += ay;
        }
        if (len > t0 || bd.chunks.empty()) bd.chunks.push_back(StreamChunkDef{{StreamPiece{I, t0, len}}});
      }
    }
  }
}

}  // namespace bsramg
