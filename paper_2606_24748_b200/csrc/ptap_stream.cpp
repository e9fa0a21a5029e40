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
#include <cstring>
#include <numeric>
#include <queue>

#include "internal.h"

namespace bsramg {

static inline int64_t up16(int64_t b) { return (b + 15) & ~int64_t(15); }

int64_t stream_smem_bytes(const StreamShape& sh, int ngroups, bool wide, int64_t nx, int64_t ny, int64_t ncodes,
                          int64_t nitems, int64_t nparts, int64_t nacc) {
  int64_t b = 0;
  b += up16(nacc * sh.M * sh.N * 8);
  b += up16(nx * stream_xs(sh.M, sh.K) * 8);
  b += up16(ny * sh.K * sh.N * 8);
  b += up16(nparts * sh.M * sh.N * 8);
  b += up16(ncodes * (wide ? 4 : 2));
  b += up16(nitems * (int64_t)sizeof(StreamItem));
  b += up16((int64_t)(ngroups + 1) * 4);
  return b;
}

namespace {

struct LocalChunk {
  std::vector<StreamRun> xruns, yruns;
  std::vector<StreamItem> items;
  std::vector<int32_t> gptr;
  std::vector<StreamRed> reds;
  std::vector<uint32_t> ox, yi;  // per product (unpacked)
  int32_t nx = 0, ny = 0, nparts = 0;
};
struct LocalBrick {
  std::vector<LocalChunk> chunks;
  std::vector<int32_t> acc_slot;
  uint32_t max_ox = 0, max_yi = 0;
  bool bad = false;
};

}  // namespace

void stream_build(const StreamShape& sh, int ngroups, int max_item, int64_t smem_budget,
                  const std::vector<StreamBrickDef>& bricks, const int32_t* rowptr_x, const int32_t* colidx_x,
                  const int32_t* rowptr_y, const int32_t* rowptr_c, const int32_t* pairptr, const uint16_t* off_x,
                  const uint16_t* off_y, StreamPlan& out) {
  out = StreamPlan();
  out.ngroups = ngroups;
  const int64_t nb = (int64_t)bricks.size();
  std::vector<LocalBrick> L((size_t)nb);
  if (max_item < 1) max_item = 1;
  if (max_item > 65535) max_item = 65535;

#pragma omp parallel
  {
    std::vector<int32_t> ycols, ydst, order, load_of;
#pragma omp for schedule(dynamic, 16)
    for (int64_t b = 0; b < nb; ++b) {
      const StreamBrickDef& bd = bricks[(size_t)b];
      LocalBrick& lb = L[(size_t)b];
      // accumulator entries: every C slot of every distinct row of the brick (accumulate mode only)
      std::vector<int32_t> rows;
      std::vector<int32_t> acc_base;
      if (!bd.direct) {
        for (const auto& cd : bd.chunks)
          for (const auto& pc : cd.pieces) rows.push_back(pc.row);
        std::sort(rows.begin(), rows.end());
        rows.erase(std::unique(rows.begin(), rows.end()), rows.end());
        acc_base.resize(rows.size());
        for (size_t r = 0; r < rows.size(); ++r) {
          acc_base[r] = (int32_t)lb.acc_slot.size();
          for (int32_t s = rowptr_c[rows[r]]; s < rowptr_c[rows[r] + 1]; ++s) lb.acc_slot.push_back(s);
        }
      }
      lb.chunks.resize(bd.chunks.size());
      for (size_t ci = 0; ci < bd.chunks.size(); ++ci) {
        const StreamChunkDef& cd = bd.chunks[ci];
        LocalChunk& lc = lb.chunks[ci];
        // ---- X runs and the Y rows they reference
        std::vector<int32_t> piece_xbase(cd.pieces.size());
        ycols.clear();
        int32_t dst = 0;
        for (size_t pi = 0; pi < cd.pieces.size(); ++pi) {
          const StreamPiece& pc = cd.pieces[pi];
          const int32_t src = rowptr_x[pc.row] + pc.t0, n = pc.t1 - pc.t0;
          piece_xbase[pi] = dst;
          if (n <= 0) continue;
          if (!lc.xruns.empty() && lc.xruns.back().src + lc.xruns.back().n == src) lc.xruns.back().n += n;
          else lc.xruns.push_back({src, n, dst});
          for (int32_t k = src; k < src + n; ++k) ycols.push_back(colidx_x[k]);
          dst += n;
        }
        lc.nx = dst;
        std::sort(ycols.begin(), ycols.end());
        ycols.erase(std::unique(ycols.begin(), ycols.end()), ycols.end());
        ydst.resize(ycols.size());
        int32_t yd = 0;
        for (size_t t = 0; t < ycols.size(); ++t) {
          const int32_t j = ycols[t], src = rowptr_y[j], n = rowptr_y[j + 1] - rowptr_y[j];
          ydst[t] = yd;
          if (n > 0) {
            if (!lc.yruns.empty() && lc.yruns.back().src + lc.yruns.back().n == src) lc.yruns.back().n += n;
            else lc.yruns.push_back({src, n, yd});
          }
          yd += n;
        }
        lc.ny = yd;
        // ---- items (slot-major; a slot's products inside one piece are contiguous because off_x ascends)
        for (size_t pi = 0; pi < cd.pieces.size(); ++pi) {
          const StreamPiece& pc = cd.pieces[pi];
          if (pc.t1 <= pc.t0) continue;
          const size_t racc = bd.direct ? 0 : (size_t)(std::lower_bound(rows.begin(), rows.end(), pc.row) - rows.begin());
          for (int32_t s = rowptr_c[pc.row]; s < rowptr_c[pc.row + 1]; ++s) {
            const uint16_t* ob = off_x + pairptr[s];
            const uint16_t* oe = off_x + pairptr[s + 1];
            const int64_t a = pairptr[s] + (std::lower_bound(ob, oe, (uint16_t)pc.t0) - ob);
            const int64_t e = (pc.t1 > 0xffff) ? pairptr[s + 1]
                                               : pairptr[s] + (std::lower_bound(ob, oe, (uint16_t)pc.t1) - ob);
            if (e <= a) continue;
            const int32_t part_first = lc.nparts;
            for (int64_t p = a; p < e;) {
              const int32_t n = (int32_t)std::min<int64_t>(bd.direct ? 65535 : max_item, e - p);
              StreamItem it;
              it.p0 = (int32_t)lc.ox.size();
              it.n = (uint16_t)n;
              if (piece_xbase[pi] > 0xffff) lb.bad = true;
              it.xrow = (uint16_t)piece_xbase[pi];
              if (bd.direct) {
                if (p != a || n != e - a || pc.t0 != 0) lb.bad = true;  // a direct block must be one item
                it.out = s;
              } else {
                it.out = -(lc.nparts++) - 1;
              }
              for (int64_t q = p; q < p + n; ++q) {
                const uint32_t ox = off_x[q];
                const int32_t j = colidx_x[rowptr_x[pc.row] + ox];
                const size_t t = (size_t)(std::lower_bound(ycols.begin(), ycols.end(), j) - ycols.begin());
                const uint32_t oxr = ox - (uint32_t)pc.t0, yi = (uint32_t)ydst[t] + off_y[q];
                lc.ox.push_back(oxr);
                lc.yi.push_back(yi);
                lb.max_ox = std::max(lb.max_ox, oxr);
                lb.max_yi = std::max(lb.max_yi, yi);
              }
              lc.items.push_back(it);
              p += n;
            }
            if (!bd.direct)
              lc.reds.push_back({acc_base[racc] + (s - rowptr_c[pc.row]), part_first, lc.nparts - part_first});
          }
        }
        // ---- schedule: longest item first onto the least loaded lane group, then store the items group-major
        const size_t ni = lc.items.size();
        order.resize(ni);
        std::iota(order.begin(), order.end(), 0);
        std::stable_sort(order.begin(), order.end(),
                         [&](int32_t u, int32_t v) { return lc.items[(size_t)u].n > lc.items[(size_t)v].n; });
        typedef std::pair<int64_t, int32_t> LG;  // (load, group)
        std::priority_queue<LG, std::vector<LG>, std::greater<LG>> pq;
        for (int g = 0; g < ngroups; ++g) pq.push({0, g});
        load_of.assign(ni, 0);
        std::vector<int32_t> cnt((size_t)ngroups + 1, 0);
        for (size_t t = 0; t < ni; ++t) {
          LG top = pq.top();
          pq.pop();
          load_of[(size_t)order[t]] = top.second;
          cnt[(size_t)top.second + 1]++;
          top.first += lc.items[(size_t)order[t]].n + 3;  // + per-item overhead (fetch, flush)
          pq.push(top);
        }
        for (int g = 0; g < ngroups; ++g) cnt[(size_t)g + 1] += cnt[(size_t)g];
        lc.gptr = cnt;
        std::vector<StreamItem> sorted(ni);
        std::vector<int32_t> fill(cnt.begin(), cnt.end() - 1);
        for (size_t t = 0; t < ni; ++t) sorted[(size_t)fill[(size_t)load_of[(size_t)order[t]]]++] = lc.items[(size_t)order[t]];
        lc.items.swap(sorted);
      }
    }
  }
  // ---- code width and limits
  uint32_t max_ox = 0, max_yi = 0;
  for (const auto& lb : L) {
    if (lb.bad) { out.why = "brick outside the stream format"; return; }
    max_ox = std::max(max_ox, lb.max_ox);
    max_yi = std::max(max_yi, lb.max_yi);
  }
  if (max_ox < 32 && max_yi < 2048) { out.wide = false; out.oxbits = 5; }
  else if (max_ox < 4096 && max_yi < (1u << 20)) { out.wide = true; out.oxbits = 12; }
  else { out.why = "row or staged operand too long for the product codes"; return; }
  // ---- flatten
  int64_t nchunks = 0, nacc = 0;
  for (const auto& lb : L) { nchunks += (int64_t)lb.chunks.size(); nacc += (int64_t)lb.acc_slot.size(); }
  out.br_chunk_ptr.resize((size_t)nb + 1);
  out.br_acc_ptr.resize((size_t)nb + 1);
  out.acc_slot.reserve((size_t)nacc);
  out.ch_xrun_ptr.assign((size_t)nchunks + 1, 0);
  out.ch_yrun_ptr.assign((size_t)nchunks + 1, 0);
  out.ch_item_ptr.assign((size_t)nchunks + 1, 0);
  out.ch_red_ptr.assign((size_t)nchunks + 1, 0);
  out.ch_code_ptr.assign((size_t)nchunks + 1, 0);
  out.ch_gptr.resize((size_t)nchunks * (ngroups + 1));
  out.ch_nx.resize((size_t)nchunks);
  out.ch_ny.resize((size_t)nchunks);
  out.ch_nparts.resize((size_t)nchunks);
  int64_t c = 0, nxr = 0, nyr = 0, nit = 0, nrd = 0, ncd = 0;
  for (int64_t b = 0; b < nb; ++b) {
    const LocalBrick& lb = L[(size_t)b];
    out.br_chunk_ptr[(size_t)b] = (int32_t)c;
    out.br_acc_ptr[(size_t)b] = (int32_t)out.acc_slot.size();
    out.acc_slot.insert(out.acc_slot.end(), lb.acc_slot.begin(), lb.acc_slot.end());
    for (const auto& lc : lb.chunks) {
      out.ch_xrun_ptr[(size_t)c] = (int32_t)nxr; out.ch_yrun_ptr[(size_t)c] = (int32_t)nyr;
      out.ch_item_ptr[(size_t)c] = (int32_t)nit; out.ch_red_ptr[(size_t)c] = (int32_t)nrd;
      out.ch_code_ptr[(size_t)c] = ncd;
      out.ch_nx[(size_t)c] = lc.nx; out.ch_ny[(size_t)c] = lc.ny; out.ch_nparts[(size_t)c] = lc.nparts;
      std::copy(lc.gptr.begin(), lc.gptr.end(), out.ch_gptr.begin() + c * (ngroups + 1));
      const int64_t smem = stream_smem_bytes(sh, ngroups, out.wide, lc.nx, lc.ny, (int64_t)lc.ox.size(),
                                             (int64_t)lc.items.size(), lc.nparts, (int64_t)lb.acc_slot.size());
      out.max_smem = std::max(out.max_smem, smem);
      nxr += (int64_t)lc.xruns.size(); nyr += (int64_t)lc.yruns.size(); nit += (int64_t)lc.items.size();
      nrd += (int64_t)lc.reds.size(); ncd += (int64_t)lc.ox.size();
      ++c;
    }
  }
  out.br_chunk_ptr[(size_t)nb] = (int32_t)c;
  out.br_acc_ptr[(size_t)nb] = (int32_t)out.acc_slot.size();
  out.ch_xrun_ptr[(size_t)c] = (int32_t)nxr; out.ch_yrun_ptr[(size_t)c] = (int32_t)nyr;
  out.ch_item_ptr[(size_t)c] = (int32_t)nit; out.ch_red_ptr[(size_t)c] = (int32_t)nrd;
  out.ch_code_ptr[(size_t)c] = ncd;
  if (nit >= (1LL << 31) || out.max_smem > smem_budget) {
    out.why = out.max_smem > smem_budget ? "a brick does not fit the shared memory budget" : "too many items";
    return;
  }
  out.xruns.resize((size_t)nxr); out.yruns.resize((size_t)nyr); out.items.resize((size_t)nit);
  out.reds.resize((size_t)nrd);
  if (out.wide) out.codes32.resize((size_t)ncd); else out.codes16.resize((size_t)ncd);
  const int oxb = out.oxbits;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t b = 0; b < nb; ++b) {
    const LocalBrick& lb = L[(size_t)b];
    int64_t cc = out.br_chunk_ptr[(size_t)b];
    for (const auto& lc : lb.chunks) {
      std::copy(lc.xruns.begin(), lc.xruns.end(), out.xruns.begin() + out.ch_xrun_ptr[(size_t)cc]);
      std::copy(lc.yruns.begin(), lc.yruns.end(), out.yruns.begin() + out.ch_yrun_ptr[(size_t)cc]);
      std::copy(lc.items.begin(), lc.items.end(), out.items.begin() + out.ch_item_ptr[(size_t)cc]);
      std::copy(lc.reds.begin(), lc.reds.end(), out.reds.begin() + out.ch_red_ptr[(size_t)cc]);
      const int64_t c0 = out.ch_code_ptr[(size_t)cc];
      for (size_t p = 0; p < lc.ox.size(); ++p) {
        const uint32_t code = lc.ox[p] | (lc.yi[p] << oxb);
        if (out.wide) out.codes32[(size_t)c0 + p] = code; else out.codes16[(size_t)c0 + p] = (uint16_t)code;
      }
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
void stream_bricks_stage1(const HostPlan& hp, const StreamShape& sh, int ngroups, int64_t smem_budget,
                          const int32_t* rowptr_a, const int32_t* colidx_a, const int32_t* rowptr_p,
                          std::vector<StreamBrickDef>& bricks) {
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
        int64_t nx = 0, ny = 0, ncodes = 0, nitems = 0;
        cols.clear();
        for (int32_t t = r.first; t < r.second; ++t) {
          const int32_t i = grows[t];
          nx += rowptr_a[i + 1] - rowptr_a[i];
          nitems += hp.rowptr_ap[i + 1] - hp.rowptr_ap[i];
          ncodes += hp.pairptr1[hp.rowptr_ap[i + 1]] - hp.pairptr1[hp.rowptr_ap[i]];
          cols.insert(cols.end(), colidx_a + rowptr_a[i], colidx_a + rowptr_a[i + 1]);
        }
        std::sort(cols.begin(), cols.end());
        cols.erase(std::unique(cols.begin(), cols.end()), cols.end());
        for (int32_t j : cols) ny += rowptr_p[j + 1] - rowptr_p[j];
        const int64_t bytes = stream_smem_bytes(sh, ngroups, /*wide=*/ny >= 2048, nx, ny, ncodes, nitems, 0, 0);
        if (bytes > smem_budget && r.second - r.first > 1) {
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
void stream_bricks_stage2(const HostPlan& hp, const StreamShape& sh, int ngroups, int max_item, int64_t smem_budget,
                          const int32_t* rowptr_r, const int32_t* colidx_r, std::vector<StreamBrickDef>& bricks) {
  const int32_t nc = hp.nbcols_p;
  bricks.assign((size_t)nc, StreamBrickDef());
#pragma omp parallel
  {
    std::vector<int32_t> cnt;
#pragma omp for schedule(dynamic, 64)
    for (int32_t I = 0; I < nc; ++I) {
      StreamBrickDef& bd = bricks[(size_t)I];
      bd.direct = false;
      const int32_t len = rowptr_r[I + 1] - rowptr_r[I];
      const int64_t nslots = hp.rowptr_c[I + 1] - hp.rowptr_c[I];
      cnt.assign((size_t)len + 1, 0);
      for (int64_t p = hp.pairptr2[hp.rowptr_c[I]]; p < hp.pairptr2[hp.rowptr_c[I + 1]]; ++p) cnt[hp.t2[(size_t)p]]++;
      int32_t t0 = 0;
      int64_t nx = 0, ny = 0, ncodes = 0;
      for (int32_t t = 0; t < len; ++t) {
        const int32_t i = colidx_r[rowptr_r[I] + t];
        const int64_t ay = hp.rowptr_ap[i + 1] - hp.rowptr_ap[i], ac = cnt[(size_t)t];
        const int64_t est_items = nslots + (ncodes + ac) / std::max(1, max_item);
        const int64_t bytes = stream_smem_bytes(sh, ngroups, true, nx + 1, ny + ay, ncodes + ac, est_items, est_items, nslots);
        if (bytes > smem_budget && t > t0) {
          bd.chunks.push_back(StreamChunkDef{{StreamPiece{I, t0, t}}});
          t0 = t; nx = 0; ny = 0; ncodes = 0;
        }
        nx += 1; ny += ay; ncodes += ac;
      }
      if (len > t0 || bd.chunks.empty()) bd.chunks.push_back(StreamChunkDef{{StreamPiece{I, t0, len}}});
    }
  }
}

}  // namespace bsramg
