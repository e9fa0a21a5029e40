// ptap_prog.cpp -- host side (cold) of the numeric PtAP: builds the lane programs of ptap_prog.h.
//
// the blocked COO plan is built once ("coordinates declared once", duplicate-summation map)
// and every numeric assembly reuses it.  Here the map is a program per brick: which lane multiplies which staged
// blocks in which order and where each output block is written, so the hot kernels (ptap_prog.cu) search nothing and
// use no atomics.  PAPER.md:103, 219: stage 1 is the dominant fine-level product AP = A*P, stage 2 the R*(AP) product.
//
// Integer work only; OpenMP over bricks; nothing here runs in the hot calls.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <numeric>
#include <unordered_map>

#include "internal.h"
#include "ptap_prog.h"

namespace bsramg {

namespace {

inline int64_t up16(int64_t b) { return (b + 15) & ~int64_t(15); }

inline uint64_t mix64(uint64_t h, uint64_t v) {
  h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2);
  h *= 0xff51afd7ed558ccdull;
  return h ^ (h >> 33);
}

struct Prod { int32_t x, yrow, q; };   // X block (index over the brick's concatenated rows), staged Y row, block in it
struct Item {
  int32_t r, t, col;
  std::vector<Prod> prods;             // ascending X block = ascending inner index
};

// all output blocks of a brick with their products, from the relative structure
void make_items(const RelBrick& rb, std::vector<Item>& items, std::vector<int32_t>& xoff, std::vector<int32_t>& yoff) {
  const int32_t nrows = (int32_t)rb.xlen.size(), nyrows = (int32_t)rb.ylen.size();
  xoff.assign((size_t)nrows + 1, 0);
  yoff.assign((size_t)nyrows + 1, 0);
  for (int32_t r = 0; r < nrows; ++r) xoff[(size_t)r + 1] = xoff[r] + rb.xlen[r];
  for (int32_t y = 0; y < nyrows; ++y) yoff[(size_t)y + 1] = yoff[y] + rb.ylen[y];
  items.clear();
  std::vector<int32_t> where((size_t)rb.ncols, -1);
  int32_t coff = 0;
  for (int32_t r = 0; r < nrows; ++r) {
    const size_t first = items.size();
    for (int32_t t = 0; t < rb.clen[r]; ++t) {
      const int32_t c = rb.ccol[(size_t)coff + t];
      where[c] = (int32_t)items.size();
      items.push_back(Item{r, t, c, {}});
    }
    for (int32_t k = 0; k < rb.xlen[r]; ++k) {
      const int32_t x = xoff[r] + k, y = rb.xcol[x];
      for (int32_t q = 0; q < rb.ylen[y]; ++q) {
        const int32_t w = where[rb.ycol[(size_t)yoff[y] + q]];
        if (w >= (int32_t)first) items[(size_t)w].prods.push_back(Prod{x, y, q});
      }
    }
    for (size_t s = first; s < items.size(); ++s) where[items[s].col] = -1;
    coff += rb.clen[r];
  }
}

// a (virtual) output column: the items it owns.  A column heavier than one class's share is cut into several
// virtual columns (their Y blocks are then staged once per class that needs them).
struct VCol { int64_t w = 0; std::vector<int32_t> items; int cls = -1; };

// longest-processing-time assignment of weights to `nbins` bins; returns bin per entry
std::vector<int> lpt(const std::vector<int64_t>& w, int nbins, const std::vector<int>* maxcount = nullptr) {
  std::vector<int32_t> order(w.size());
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return w[a] > w[b]; });
  std::vector<int64_t> load((size_t)nbins, 0);
  std::vector<int> cnt((size_t)nbins, 0), bin(w.size(), 0);
  for (int32_t e : order) {
    int best = -1;
    for (int b = 0; b < nbins; ++b) {
      if (maxcount && cnt[b] >= (*maxcount)[b]) continue;
      if (best < 0 || load[b] < load[best]) best = b;
    }
    if (best < 0) best = 0;
    bin[e] = best;
    load[best] += w[e];
    cnt[best]++;
  }
  return bin;
}

inline uint32_t mkdesc(int32_t xs, int32_t ys, int flag) { return (uint32_t)xs | ((uint32_t)ys << 12) | ((uint32_t)flag << 24); }
inline int lane_of(int cls, int m) { return (m / 4) * 32 + cls + 8 * (m % 4); }   // m-th lane of a class -> thread id

// Y slots of one chunk: the blocks each class reads, slot = 8 * index + class.  Index 0 of every class is a zero block
// (written by the kernel): padding steps multiply the zero X block with it, so they read initialised, conflict-free
// shared memory and add exact zeros.
struct YSlots {
  std::vector<YCopy> copies;
  std::unordered_map<uint64_t, int32_t> slot;   // (class, yrow, q) -> slot
  int32_t count[PROG_NCLASS] = {0, 0, 0, 0, 0, 0, 0, 0};
  int32_t get(int cls, int32_t yrow, int32_t q) {
    const uint64_t key = ((uint64_t)cls << 48) | ((uint64_t)(uint32_t)yrow << 20) | (uint64_t)(uint32_t)q;
    auto it = slot.find(key);
    if (it != slot.end()) return it->second;
    const int32_t s = 8 * (++count[cls]) + cls;
    slot.emplace(key, s);
    copies.push_back(YCopy{(uint16_t)yrow, (uint16_t)q, (uint16_t)s, 0});
    return s;
  }
  int32_t nslots() const { return 8 * (1 + *std::max_element(count, count + PROG_NCLASS)); }
};

}  // namespace

uint64_t RelBrick::hash() const {
  uint64_t h = 0x243f6a8885a308d3ull;
  auto feed = [&](const std::vector<int32_t>& v) {
    h = mix64(h, v.size());
    for (int32_t e : v) h = mix64(h, (uint64_t)(uint32_t)e);
  };
  feed(xlen); feed(xcol); feed(ylen); feed(ycol); feed(clen); feed(ccol);
  return h;
}

int64_t prog_blob_words(bool persist, bool last_chunk, int32_t nrows, int32_t nfix, const ProgChunk& ch) {
  int64_t w = PROG_H_WORDS + 2 * (int64_t)ch.nxrun + ch.nycopy;
  w = (w + 3) & ~int64_t(3);
  w += ch.blob_words;
  if (last_chunk) w += nrows + 2 * (int64_t)nfix + (persist ? PROG_NT : 0);
  return (w + 3) & ~int64_t(3);
}

ProgSmem prog_smem_bytes(const ProgShape& sh, bool persist, bool last_chunk, int32_t nrows, int32_t nyrows, int32_t nfix,
                         int32_t ncs_all, const ProgChunk& ch) {
  ProgSmem m;
  m.rec = (int64_t)prog_rec_words(nrows, nyrows) * 4;
  m.blob = prog_blob_words(persist, last_chunk, nrows, nfix, ch) * 4;
  m.xy = up16((int64_t)(ch.nx + 8) * prog_xs(sh) * 8) + (int64_t)ch.nyslots * prog_yc16(sh) * 16;
  m.low = 3 * m.rec + 2 * m.blob + m.xy;   // record ring, this blob and the prefetched next one, operands
  m.cs = up16((int64_t)ncs_all * sh.M * sh.N * 8);
  return m;
}

namespace {

// One lane's work inside one warp program: segments of products that are accumulated into one staged block.  A segment
// occupies whole rounds; `store` is the staging slot written at the end of its last round (PROG_NONE: persist mode).
struct Seg { std::vector<Prod> prods; int32_t rounds; uint32_t store; };

// Orders the products of every segment over the steps of its rounds so that the eight lanes of a quarter warp read
// X slots in eight different 16-byte bank groups whenever they can (the Y slots are conflict free by class), and
// emits the warp's program words.  Returns the number of rounds.
int emit_warp(const ProgShape& sh, int w, int G, bool with_store, int32_t nx, const std::vector<std::vector<Seg>>& lane_segs,
              const std::vector<std::vector<std::vector<int32_t>>>& yslot, std::vector<uint32_t>& blob) {
  const int xc16 = prog_xs(sh) / 2;
  int rounds = 0;
  for (int l = 0; l < 32; ++l) {
    int r = 0;
    for (const Seg& sg : lane_segs[(size_t)w * 32 + l]) r += sg.rounds;
    rounds = std::max(rounds, r);
  }
  // per lane: which segment is active in which round
  std::vector<std::vector<int32_t>> seg_of((size_t)32, std::vector<int32_t>((size_t)rounds, -1));
  std::vector<std::vector<int32_t>> last_round((size_t)32);
  for (int l = 0; l < 32; ++l) {
    int r = 0;
    const auto& segs = lane_segs[(size_t)w * 32 + l];
    for (size_t g = 0; g < segs.size(); ++g) {
      for (int k = 0; k < segs[g].rounds; ++k) seg_of[l][(size_t)r + k] = (int32_t)g;
      r += segs[g].rounds;
      last_round[l].push_back(r - 1);
    }
  }
  std::vector<std::vector<std::vector<char>>> used((size_t)32);
  for (int l = 0; l < 32; ++l) {
    const auto& segs = lane_segs[(size_t)w * 32 + l];
    used[l].resize(segs.size());
    for (size_t g = 0; g < segs.size(); ++g) used[l][g].assign(segs[g].prods.size(), 0);
  }
  std::vector<std::vector<int32_t>> left((size_t)32);   // steps left in the segment (to know when padding is allowed)
  for (int l = 0; l < 32; ++l) {
    const auto& segs = lane_segs[(size_t)w * 32 + l];
    for (const Seg& sg : segs) left[l].push_back(sg.rounds * G);
  }
  std::vector<std::vector<int32_t>> remaining((size_t)32);
  for (int l = 0; l < 32; ++l)
    for (const Seg& sg : lane_segs[(size_t)w * 32 + l]) remaining[l].push_back((int32_t)sg.prods.size());
  for (int r = 0; r < rounds; ++r) {
    for (int s = 0; s < G; ++s) {
      uint32_t row[32];
      for (int qd = 0; qd < 4; ++qd) {
        int taken[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // lanes already reading a (different) X slot in this bank group
        int32_t slot_in_group[8] = {-1, -1, -1, -1, -1, -1, -1, -1};
        // lanes that must take a product now (no slack left) first, then the others
        int order[8], n = 0;
        for (int pass = 0; pass < 2; ++pass)
          for (int a = 0; a < 8; ++a) {
            const int l = qd * 8 + a;
            const int32_t g = seg_of[l][(size_t)r];
            const bool must = g >= 0 && remaining[l][(size_t)g] >= left[l][(size_t)g];
            if ((pass == 0) == must) order[n++] = a;
          }
        for (int oi = 0; oi < 8; ++oi) {
          const int a = order[oi], l = qd * 8 + a;
          const int32_t g = seg_of[l][(size_t)r];
          int32_t pick = -1;
          if (g >= 0 && remaining[l][(size_t)g] > 0) {
            const Seg& sg = lane_segs[(size_t)w * 32 + l][(size_t)g];
            int best = 1 << 30;
            for (size_t p = 0; p < sg.prods.size(); ++p) {
              if (used[l][(size_t)g][p]) continue;
              const int grp = (sg.prods[p].x * xc16) & 7;
              const int cost = slot_in_group[grp] == sg.prods[p].x ? 0 : taken[grp];
              if (cost < best) { best = cost; pick = (int32_t)p; if (cost == 0) break; }
            }
            // a conflicting pick can wait if the segment still has slack (a padding step now, the product later)
            if (best > 0 && remaining[l][(size_t)g] < left[l][(size_t)g]) pick = -1;
          }
          if (pick >= 0) {
            const Seg& sg = lane_segs[(size_t)w * 32 + l][(size_t)g];
            const Prod& pr = sg.prods[(size_t)pick];
            used[l][(size_t)g][(size_t)pick] = 1;
            remaining[l][(size_t)g]--;
            const int grp = (pr.x * xc16) & 7;
            if (slot_in_group[grp] != pr.x) { taken[grp]++; slot_in_group[grp] = pr.x; }
            row[l] = mkdesc(pr.x, yslot[(size_t)w * 32 + l][(size_t)g][(size_t)pick], 0);
          } else {
            // padding: one of the eight zero X blocks (consecutive slots = eight different bank groups), free if any
            int z = 0, bestz = 1 << 30;
            for (int k = 0; k < 8; ++k) {
              const int grp = ((nx + k) * xc16) & 7;
              const int cost = slot_in_group[grp] == nx + k ? 0 : taken[grp];
              if (cost < bestz) { bestz = cost; z = k; }
            }
            const int grp = ((nx + z) * xc16) & 7;
            if (slot_in_group[grp] != nx + z) { taken[grp]++; slot_in_group[grp] = nx + z; }
            row[l] = mkdesc(nx + z, l & 7, 0);
          }
          if (g >= 0) left[l][(size_t)g]--;
        }
      }
      blob.insert(blob.end(), row, row + 32);
    }
    if (with_store)
      for (int l = 0; l < 32; ++l) {
        const int32_t g = seg_of[l][(size_t)r];
        uint32_t sw = PROG_NONE;
        if (g >= 0 && last_round[l][(size_t)g] == r) sw = lane_segs[(size_t)w * 32 + l][(size_t)g].store;
        blob.push_back(sw);
      }
  }
  return rounds;
}

}  // namespace

// ------------------------------------------------------------------ direct programs (stage 1)
static void build_direct(const ProgShape& sh, int G, const RelBrick& rb, Program& out) {
  std::vector<Item> items;
  std::vector<int32_t> xoff, yoff;
  make_items(rb, items, xoff, yoff);
  const int32_t nrows = (int32_t)rb.xlen.size(), nx = xoff[nrows];
  if (nx > 4080 || nrows > 65535 || (int32_t)rb.ylen.size() > 65535) { out.why = "brick has too many X blocks"; return; }
  std::vector<int32_t> coff((size_t)nrows + 1, 0);
  for (int32_t r = 0; r < nrows; ++r) {
    if (rb.clen[r] > 65535 || rb.xlen[r] > 65535) { out.why = "row too long"; return; }
    coff[(size_t)r + 1] = coff[r] + rb.clen[r];
  }
  const int32_t ncs = coff[nrows];
  auto nslots = [&](const Item& it) { return (int64_t)((it.prods.size() + (size_t)G - 1) / (size_t)G); };
  // ---- virtual columns and classes, balanced in slots (a slot = one round of one lane)
  int64_t total = 0, total_slots = 0;
  std::vector<std::vector<int32_t>> by_col((size_t)rb.ncols);
  for (size_t s = 0; s < items.size(); ++s) {
    by_col[(size_t)items[s].col].push_back((int32_t)s);
    total += (int64_t)items[s].prods.size();
    total_slots += nslots(items[s]);
  }
  const int64_t cap = std::max<int64_t>(1, (total_slots + PROG_NCLASS - 1) / PROG_NCLASS);
  std::vector<VCol> vcols;
  for (auto& list : by_col) {
    if (list.empty()) continue;
    int64_t w = 0;
    for (int32_t s : list) w += nslots(items[(size_t)s]);
    const int nsplit = (int)std::min<int64_t>((w + cap - 1) / cap, (int64_t)list.size());
    int64_t acc = 0;
    int part = 0;
    vcols.push_back(VCol());
    for (int32_t s : list) {
      const int64_t ws = nslots(items[(size_t)s]);
      if (part + 1 < nsplit && acc > 0 && acc + ws / 2 > (w * (part + 1)) / nsplit) {
        vcols.push_back(VCol());
        ++part;
      }
      vcols.back().items.push_back(s);
      vcols.back().w += ws;
      acc += ws;
    }
  }
  {
    // classes balanced in slots (time) first and in staged Y blocks (shared memory: every class gets as many Y
    // slots as the fullest one) second
    std::vector<int64_t> w(vcols.size()), yb(vcols.size(), 0);
    int64_t ytot = 0;
    for (size_t v = 0; v < vcols.size(); ++v) {
      w[v] = vcols[v].w;
      std::vector<uint64_t> blocks;
      for (int32_t s : vcols[v].items)
        for (const Prod& pr : items[(size_t)s].prods) blocks.push_back(((uint64_t)(uint32_t)pr.yrow << 20) | (uint32_t)pr.q);
      std::sort(blocks.begin(), blocks.end());
      yb[v] = (int64_t)(std::unique(blocks.begin(), blocks.end()) - blocks.begin());
      ytot += yb[v];
    }
    std::vector<int32_t> order(vcols.size());
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return w[a] > w[b]; });
    int64_t lw[PROG_NCLASS] = {0}, ly[PROG_NCLASS] = {0};
    for (int32_t v : order) {
      int best = 0;
      double bestcost = 1e300;
      for (int c = 0; c < PROG_NCLASS; ++c) {
        const double cw = (double)(lw[c] + w[(size_t)v]) / (double)std::max<int64_t>(1, total_slots);
        const double cy = (double)(ly[c] + yb[(size_t)v]) / (double)std::max<int64_t>(1, ytot);
        const double cost = std::max(cw, 0.85 * cy) + 0.05 * cw;
        if (cost < bestcost) { bestcost = cost; best = c; }
      }
      vcols[(size_t)v].cls = best;
      lw[best] += w[(size_t)v]; ly[best] += yb[(size_t)v];
    }
  }
  // ---- lanes: every class has PROG_LPC lanes and needs R = ceil(slots / lanes) rounds.  Items go to the lane with
  // the most room, largest first; an item that fits nowhere in one piece is cut into parts on several lanes (its
  // later parts go to overflow slots and are added to the first part before the rows are written)
  YSlots ys;
  std::vector<std::vector<Seg>> lane_segs((size_t)PROG_NT);
  std::vector<std::vector<std::vector<int32_t>>> yslot((size_t)PROG_NT);
  std::vector<int32_t> nparts(items.size(), 0), ovf_first(items.size(), -1);
  struct PartRef { int32_t t; size_t seg; int32_t item, part; };
  std::vector<PartRef> later_parts;
  for (int c = 0; c < PROG_NCLASS; ++c) {
    std::vector<int32_t> cit;
    for (const VCol& v : vcols)
      if (v.cls == c) cit.insert(cit.end(), v.items.begin(), v.items.end());
    int64_t S = 0;
    for (int32_t s : cit) S += nslots(items[(size_t)s]);
    if (S == 0) continue;
    const int64_t R = (S + PROG_LPC - 1) / PROG_LPC;
    std::stable_sort(cit.begin(), cit.end(), [&](int32_t a, int32_t b) { return items[(size_t)a].prods.size() > items[(size_t)b].prods.size(); });
    int64_t room[PROG_LPC];
    for (int m = 0; m < PROG_LPC; ++m) room[m] = R;
    auto give = [&](int32_t s, int m, int64_t slot0, int64_t take) {
      const Item& it = items[(size_t)s];
      Seg sg;
      const size_t p0 = (size_t)slot0 * (size_t)G, p1 = std::min(it.prods.size(), (size_t)(slot0 + take) * (size_t)G);
      sg.prods.assign(it.prods.begin() + (std::ptrdiff_t)p0, it.prods.begin() + (std::ptrdiff_t)p1);
      sg.rounds = (int32_t)take;
      const int32_t part = nparts[(size_t)s]++;
      sg.store = (uint32_t)(coff[it.r] + it.t);
      const int t = lane_of(c, m);
      if (part > 0) later_parts.push_back(PartRef{t, lane_segs[(size_t)t].size(), s, part});
      std::vector<int32_t> ysl;
      for (const Prod& pr : sg.prods) ysl.push_back(ys.get(c, pr.yrow, pr.q));
      lane_segs[(size_t)t].push_back(std::move(sg));
      yslot[(size_t)t].push_back(std::move(ysl));
      room[m] -= take;
    };
    for (int32_t s : cit) {
      const int64_t ns = nslots(items[(size_t)s]);
      // the lanes are visited in an order that differs per class, so that the fuller lanes of the classes spread
      // over the warps
      int best = -1;
      for (int mm = 0; mm < PROG_LPC; ++mm) {
        const int m = (mm * 5 + c * 3) % PROG_LPC;
        if (room[m] >= ns && (best < 0 || room[m] > room[best])) best = m;
      }
      if (best >= 0) { give(s, best, 0, ns); continue; }
      int64_t done = 0;
      while (done < ns) {   // no lane takes it whole: fill the lanes with the most room
        int m2 = -1;
        for (int mm = 0; mm < PROG_LPC; ++mm) {
          const int m = (mm * 5 + c * 3) % PROG_LPC;
          if (room[m] > 0 && (m2 < 0 || room[m] > room[m2])) m2 = m;
        }
        if (m2 < 0) { out.why = "internal: no room left in a class"; return; }
        const int64_t take = std::min(room[m2], ns - done);
        give(s, m2, done, take);
        done += take;
      }
    }
  }
  // overflow slots: consecutive per item, in item order; the later parts store there
  int32_t novf = 0;
  for (size_t s = 0; s < items.size(); ++s) { ovf_first[s] = novf; novf += std::max(0, nparts[s] - 1); }
  if ((int64_t)ncs + novf > 65535) { out.why = "brick has too many output blocks"; return; }
  for (const PartRef& pr : later_parts)
    lane_segs[(size_t)pr.t][pr.seg].store = (uint32_t)(ncs + ovf_first[(size_t)pr.item] + pr.part - 1);
  if (ys.nslots() > 4096) { out.why = "brick has too many Y slots"; return; }
  ProgChunk ch;
  memset(&ch, 0, sizeof ch);
  ch.xrun0 = 0; ch.nxrun = nrows;
  for (int32_t r = 0; r < nrows; ++r) out.xruns.push_back(XRun{(uint16_t)r, 0, (uint16_t)rb.xlen[r], (uint16_t)xoff[r]});
  ch.ycopy0 = 0; ch.nycopy = (int32_t)ys.copies.size();
  out.ycopies = ys.copies;
  ch.nx = nx; ch.nyslots = ys.nslots();
  ch.blob0 = 0;
  for (int w = 0; w < PROG_NW; ++w) {
    const int rounds = emit_warp(sh, w, G, true, nx, lane_segs, yslot, out.blob);
    if (rounds > 32767) { out.why = "lane list too long"; return; }
    ch.wrounds[w] = (int16_t)rounds; ch.wlen[w] = (int16_t)G;
    out.lane_steps += (int64_t)rounds * G * 32;
  }
  while (out.blob.size() & 3) out.blob.push_back(0);
  ch.blob_words = (int32_t)out.blob.size();
  out.chunks.push_back(ch);
  // tables: crow, fix
  for (int32_t r = 0; r < nrows; ++r) out.tabs.push_back((uint32_t)coff[r] | ((uint32_t)rb.clen[r] << 16));
  for (size_t s = 0; s < items.size(); ++s)
    if (nparts[s] > 1) {
      out.tabs.push_back((uint32_t)(coff[items[s].r] + items[s].t) | ((uint32_t)(ncs + ovf_first[s]) << 16));
      out.tabs.push_back((uint32_t)(nparts[s] - 1));
      out.nfix++;
    }
  out.nrows = nrows; out.nyrows = (int32_t)rb.ylen.size(); out.nout = 0;
  out.ncs = ncs; out.novf = novf;
  out.products = total;
  out.yslots_used = (int64_t)ys.copies.size();
  {
    if (out.nyrows > 4095) { out.why = "brick stages too many Y rows"; return; }
    for (const YCopy& yc : out.ycopies) if (yc.q > 255) { out.why = "row of Y too long"; return; }
    const ProgSmem m = prog_smem_bytes(sh, false, true, out.nrows, out.nyrows, out.nfix, ncs + novf, ch);
    out.smem_low = m.low; out.smem_cs = m.cs; out.smem = m.total();
    out.rec_bytes = m.rec; out.blob_bytes = m.blob; out.xy_bytes = m.xy;
  }
  out.ok = true;
  {
    // modelled shared-memory cycles of the slowest warp: 4 per 16-byte load instruction of a step, 37 per store point
    const int xl = prog_xs(sh) / 2, yl = ((sh.K * sh.N + 1) & ~1) / 2;
    int64_t worst = 0;
    for (int w = 0; w < PROG_NW; ++w) worst = std::max<int64_t>(worst, (int64_t)ch.wrounds[w] * ((int64_t)G * 4 * (xl + yl) + 4 * (sh.M * sh.N + 1) / 2 + 1));
    out.cost = worst;
  }
  if (getenv("PROG_DEBUG")) {
    int64_t cw[8] = {0};
    for (const VCol& v : vcols) cw[v.cls] += v.w;
    fprintf(stderr, "direct: rows %d nx %d items %zu total %lld slots %lld novf %d classslots", nrows, nx, items.size(),
            (long long)total, (long long)total_slots, novf);
    for (int c = 0; c < 8; ++c) fprintf(stderr, " %lld", (long long)cw[c]);
    fprintf(stderr, " rounds %d %d %d %d ycount", ch.wrounds[0], ch.wrounds[1], ch.wrounds[2], ch.wrounds[3]);
    for (int c = 0; c < 8; ++c) fprintf(stderr, " %d", ys.count[c]);
    fprintf(stderr, " smem %lld\n", (long long)out.smem);
  }
}

// ------------------------------------------------------------------ persist programs (stage 2): one row, chunks
static void build_persist(const ProgShape& sh, int64_t budget, const RelBrick& rb, Program& out) {
  if (rb.xlen.size() != 1) { out.why = "persist programs have one row"; return; }
  std::vector<Item> items;
  std::vector<int32_t> xoff, yoff;
  make_items(rb, items, xoff, yoff);
  const int32_t nx = rb.xlen[0], nyrows = (int32_t)rb.ylen.size(), nout = (int32_t)items.size();
  if (nx > 65535 || nyrows > 65535 || nout > 32767) { out.why = "row too long"; return; }
  int64_t total = 0;
  for (const Item& it : items) total += (int64_t)it.prods.size();
  // ---- virtual columns (products of a heavy column dealt round robin), classes, lanes per virtual column
  struct PV { int32_t item; int nsplit, which; int64_t w; int cls = -1; int nlanes = 0, m0 = 0; };
  std::vector<PV> pv;
  const int64_t cap = std::max<int64_t>(1, (total + PROG_NCLASS - 1) / PROG_NCLASS);
  for (int32_t s = 0; s < nout; ++s) {
    const int64_t w = (int64_t)items[(size_t)s].prods.size();
    const int ns = (int)std::max<int64_t>(1, std::min<int64_t>((w + cap - 1) / cap, w));
    for (int k = 0; k < ns; ++k) pv.push_back(PV{s, ns, k, (w - k + ns - 1) / ns});
  }
  if ((int)pv.size() > PROG_NT) { out.why = "more output columns than lanes"; return; }
  {
    std::vector<int64_t> w(pv.size());
    for (size_t v = 0; v < pv.size(); ++v) w[v] = pv[v].w;
    const std::vector<int> maxc((size_t)PROG_NCLASS, PROG_LPC);
    const std::vector<int> cls = lpt(w, PROG_NCLASS, &maxc);
    for (size_t v = 0; v < pv.size(); ++v) pv[v].cls = cls[v];
  }
  for (int c = 0; c < PROG_NCLASS; ++c) {
    std::vector<int32_t> mine;
    for (size_t v = 0; v < pv.size(); ++v)
      if (pv[v].cls == c) mine.push_back((int32_t)v);
    if (mine.empty()) continue;
    if ((int)mine.size() > PROG_LPC) { out.why = "more columns in a class than lanes"; return; }
    int left = PROG_LPC - (int)mine.size();
    for (int32_t v : mine) pv[(size_t)v].nlanes = 1;
    while (left > 0) {   // remaining lanes to whoever has the most products per lane
      int32_t best = -1;
      for (int32_t v : mine)
        if (pv[(size_t)v].nlanes < pv[(size_t)v].w &&
            (best < 0 || pv[(size_t)v].w * pv[(size_t)best].nlanes > pv[(size_t)best].w * pv[(size_t)v].nlanes)) best = v;
      if (best < 0) break;
      pv[(size_t)best].nlanes++;
      --left;
    }
    int m = 0;
    for (int32_t v : mine) { pv[(size_t)v].m0 = m; m += pv[(size_t)v].nlanes; }
  }
  // ---- every product gets its lane (round robin inside a virtual column: every chunk sees an even share)
  std::vector<std::vector<Prod>> lprods((size_t)PROG_NT);
  std::vector<std::vector<int32_t>> lanes_of_out((size_t)nout);
  for (const PV& v : pv) {
    const Item& it = items[(size_t)v.item];
    int64_t n = 0;
    for (size_t p = (size_t)v.which; p < it.prods.size(); p += (size_t)v.nsplit, ++n)
      lprods[(size_t)lane_of(v.cls, v.m0 + (int)(n % v.nlanes))].push_back(it.prods[p]);
    for (int l = 0; l < v.nlanes; ++l)
      if (!lprods[(size_t)lane_of(v.cls, v.m0 + l)].empty()) lanes_of_out[(size_t)v.item].push_back(lane_of(v.cls, v.m0 + l));
  }
  for (auto& v : lanes_of_out) {
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
  }
  int32_t novf = 0;
  for (auto& v : lanes_of_out) novf += std::max<int32_t>(0, (int32_t)v.size() - 1);
  // ---- chunks over the inner index: greedy count, then even cuts
  const int64_t fixed = 3 * (int64_t)prog_rec_words(1, nyrows) * 4;
  auto chunk_bytes = [&](int32_t k0, int32_t k1) {
    int32_t cnt[PROG_NCLASS] = {0};
    int64_t np = 0;
    for (const PV& v : pv) {
      const Item& it = items[(size_t)v.item];
      for (size_t p = (size_t)v.which; p < it.prods.size(); p += (size_t)v.nsplit)
        if (it.prods[p].x >= k0 && it.prods[p].x < k1) { cnt[v.cls]++; ++np; }
    }
    const int64_t ysl = 8 * (1 + (int64_t)*std::max_element(cnt, cnt + PROG_NCLASS));
    const int64_t blob = 2 * 4 * (np * 3 / 2 + 64 * PROG_NW + np + PROG_H_WORDS + 2 * nout + PROG_NT);
    return fixed + up16((int64_t)(k1 - k0 + 8) * prog_xs(sh) * 8) + ysl * prog_yc16(sh) * 16 + blob +
           up16((int64_t)(nout + novf) * sh.M * sh.N * 8);
  };
  for (int attempt = 0; attempt < 6; ++attempt) {
    std::vector<int32_t> cuts{0};
    {
      int32_t k0 = 0;
      for (int32_t k = 1; k <= nx; ++k)
        if (k - k0 > 1 && chunk_bytes(k0, k) > budget - attempt * 4096) { cuts.push_back(k - 1); k0 = k - 1; }
      cuts.push_back(nx);
    }
    const int nch = (int)cuts.size() - 1;
    std::vector<int64_t> pre((size_t)nx + 1, 0);
    for (const Item& it : items) for (const Prod& p : it.prods) pre[(size_t)p.x + 1]++;
    for (int32_t k = 0; k < nx; ++k) pre[(size_t)k + 1] += pre[k];
    std::vector<int32_t> ev{0};
    for (int c = 1; c < nch; ++c) {
      const int64_t target = total * c / nch;
      int32_t k = (int32_t)(std::lower_bound(pre.begin(), pre.end(), target) - pre.begin());
      k = std::max(k, ev.back() + 1);
      ev.push_back(std::min(k, nx));
    }
    ev.push_back(nx);
    bool fits = true;
    for (int c = 0; c < nch && fits; ++c) fits = ev[c + 1] > ev[c] && chunk_bytes(ev[c], ev[c + 1]) <= budget - attempt * 4096;
    const std::vector<int32_t>& use = fits ? ev : cuts;
    // ---- emit
    out.chunks.clear(); out.xruns.clear(); out.ycopies.clear(); out.blob.clear(); out.lane_steps = 0; out.yslots_used = 0;
    out.blob_bytes = 0; out.xy_bytes = 0;
    int64_t worst = 0, worst_low = 0;
    bool bad = false;
    std::vector<size_t> pos((size_t)PROG_NT, 0);
    int32_t nfix_est = 0;
    for (auto& v : lanes_of_out) nfix_est += v.size() > 1;
    for (int c = 0; c + 1 < (int)use.size(); ++c) {
      const int32_t k0 = use[c], k1 = use[c + 1];
      ProgChunk ch;
      memset(&ch, 0, sizeof ch);
      YSlots ys;
      std::vector<std::vector<Seg>> lane_segs((size_t)PROG_NT);
      std::vector<std::vector<std::vector<int32_t>>> yslot((size_t)PROG_NT);
      int maxlen[PROG_NW] = {0};
      for (int t = 0; t < PROG_NT; ++t) {
        const auto& lp = lprods[(size_t)t];
        Seg sg;
        std::vector<int32_t> ysl;
        while (pos[(size_t)t] < lp.size() && lp[pos[(size_t)t]].x < k1) {
          Prod p = lp[pos[(size_t)t]++];
          ysl.push_back(ys.get(t & 7, p.yrow, p.q));
          p.x -= k0;
          sg.prods.push_back(p);
        }
        maxlen[t / 32] = std::max(maxlen[t / 32], (int)sg.prods.size());
        sg.rounds = 1; sg.store = PROG_NONE;
        lane_segs[(size_t)t].push_back(std::move(sg));
        yslot[(size_t)t].push_back(std::move(ysl));
      }
      if (k1 - k0 > 4080 || ys.nslots() > 4096) { bad = true; break; }
      ch.xrun0 = (int32_t)out.xruns.size(); ch.nxrun = 1;
      out.xruns.push_back(XRun{0, (uint16_t)k0, (uint16_t)(k1 - k0), 0});
      ch.ycopy0 = (int32_t)out.ycopies.size(); ch.nycopy = (int32_t)ys.copies.size();
      out.ycopies.insert(out.ycopies.end(), ys.copies.begin(), ys.copies.end());
      out.yslots_used += (int64_t)ys.copies.size();
      ch.nx = k1 - k0; ch.nyslots = ys.nslots();
      ch.blob0 = (int32_t)out.blob.size();
      for (int w = 0; w < PROG_NW; ++w) {
        if (maxlen[w] > 32767) { bad = true; break; }
        ch.wrounds[w] = (int16_t)(maxlen[w] > 0 ? 1 : 0); ch.wlen[w] = (int16_t)maxlen[w];
        if (maxlen[w] > 0) emit_warp(sh, w, maxlen[w], false, k1 - k0, lane_segs, yslot, out.blob);
        out.lane_steps += (int64_t)maxlen[w] * 32;
      }
      while (out.blob.size() & 3) out.blob.push_back(0);
      ch.blob_words = (int32_t)out.blob.size() - ch.blob0;
      out.chunks.push_back(ch);
      {
        const ProgSmem m = prog_smem_bytes(sh, true, c + 2 == (int)use.size(), 1, nyrows, nfix_est, nout + novf, ch);
        out.rec_bytes = m.rec; out.blob_bytes = std::max(out.blob_bytes, m.blob); out.xy_bytes = std::max(out.xy_bytes, m.xy);
        worst = 3 * out.rec_bytes + 2 * out.blob_bytes + out.xy_bytes + m.cs;
        worst_low = worst - m.cs;
      }
    }
    if (bad) { out.why = "chunk outside the descriptor format"; return; }
    if (worst <= budget) {
      // tables: crow (one row), fix (outputs held by several lanes), pstore (staging slot of every lane)
      out.tabs.clear();
      out.tabs.push_back(0u | ((uint32_t)nout << 16));
      std::vector<uint32_t> pstore((size_t)PROG_NT, PROG_NONE);
      int32_t next = 0;
      out.nfix = 0;
      for (int32_t u = 0; u < nout; ++u) {
        const auto& ls = lanes_of_out[(size_t)u];
        if (ls.empty()) { out.why = "output block without products"; return; }
        pstore[(size_t)ls[0]] = (uint32_t)u;
        if (ls.size() > 1) {
          out.tabs.push_back((uint32_t)u | ((uint32_t)(nout + next) << 16));
          out.tabs.push_back((uint32_t)(ls.size() - 1));
          out.nfix++;
          for (size_t m = 1; m < ls.size(); ++m) pstore[(size_t)ls[m]] = (uint32_t)(nout + next++);
        }
      }
      out.tabs.insert(out.tabs.end(), pstore.begin(), pstore.end());
      out.nrows = 1; out.nyrows = nyrows; out.nout = nout;
      out.ncs = nout; out.novf = novf;
      out.products = total;
      out.smem = worst; out.smem_low = worst_low; out.smem_cs = worst - worst_low;
      if (nyrows > 4095) { out.why = "brick stages too many Y rows"; return; }
      for (const YCopy& yc : out.ycopies) if (yc.q > 255) { out.why = "row of Y too long"; return; }
      out.smem_cs = up16((int64_t)(nout + novf) * sh.M * sh.N * 8);
      out.ok = true;
      return;
    }
  }
  out.why = "row does not fit the shared-memory budget";
}

void prog_build(const ProgShape& sh, bool persist, int64_t budget, int round_len, const RelBrick& rb, Program& out) {
  out = Program();
  if (persist) build_persist(sh, budget, rb, out);
  else if (round_len > 0) build_direct(sh, round_len, rb, out);
  else {
    // round length chosen per program: the cheapest of a few candidates that fits the budget
    Program best;
    for (int G : {2, 3, 4, 5, 6, 8}) {
      Program p;
      build_direct(sh, G, rb, p);
      if (!p.ok || p.smem > budget) { if (!best.ok && best.why.empty()) best.why = p.ok ? "brick does not fit the shared-memory budget" : p.why; continue; }
      if (!best.ok || p.cost < best.cost) best = std::move(p);
    }
    out = std::move(best);
  }
  if (out.ok && out.smem > budget) { out.ok = false; out.why = "brick does not fit the shared-memory budget"; }
}

// ------------------------------------------------------------------ verification (tests; integer work only)
bool prog_verify(const ProgShape& sh, bool persist, const RelBrick& rb, const Program& p, std::string& why,
                 ProgStats* stats) {
  std::vector<Item> items;
  std::vector<int32_t> xoff, yoff;
  make_items(rb, items, xoff, yoff);
  auto fail_ = [&](const char* m) { why = m; return false; };
  if (!p.ok) return fail_("program not built");
  auto key = [](int32_t x, int32_t y, int32_t q) { return ((uint64_t)(uint32_t)x << 40) | ((uint64_t)(uint32_t)y << 16) | (uint64_t)(uint32_t)q; };
  const int32_t nrows = (int32_t)rb.xlen.size(), nslots = p.ncs + p.novf;
  std::vector<std::vector<uint64_t>> slot_prods((size_t)nslots);
  std::vector<char> slot_written((size_t)nslots, 0);
  const int xc16 = prog_xs(sh) / 2, yc16 = prog_yc16(sh);
  const uint32_t* crow = p.tabs.data();
  const uint32_t* fix = crow + nrows;
  const uint32_t* pstore = fix + 2 * (size_t)p.nfix;
  if (p.tabs.size() != (size_t)nrows + 2 * (size_t)p.nfix + (persist ? (size_t)PROG_NT : 0)) return fail_("table sizes");
  std::vector<std::vector<uint64_t>> lane_pending((size_t)PROG_NT);
  for (const ProgChunk& ch : p.chunks) {
    std::vector<int32_t> xof((size_t)ch.nx, -1);
    for (int32_t e = ch.xrun0; e < ch.xrun0 + ch.nxrun; ++e) {
      const XRun& xr = p.xruns[(size_t)e];
      if (xr.row >= rb.xlen.size() || xr.k0 + xr.n > rb.xlen[xr.row] || xr.dst + xr.n > ch.nx) return fail_("X run out of range");
      for (int32_t k = 0; k < xr.n; ++k) xof[(size_t)xr.dst + k] = xoff[xr.row] + xr.k0 + k;
    }
    std::vector<int64_t> yof((size_t)ch.nyslots, -1);
    for (int32_t e = ch.ycopy0; e < ch.ycopy0 + ch.nycopy; ++e) {
      const YCopy& yc = p.ycopies[(size_t)e];
      if (yc.slot >= ch.nyslots || yc.yrow >= rb.ylen.size() || yc.q >= rb.ylen[yc.yrow]) return fail_("Y copy out of range");
      if (yc.slot < 8) return fail_("Y copy into a zero slot");
      if (yof[yc.slot] >= 0) return fail_("Y slot written twice");
      yof[yc.slot] = ((int64_t)yc.yrow << 20) | yc.q;
    }
    const uint32_t* wd = p.blob.data() + ch.blob0;
    for (int w = 0; w < PROG_NW; ++w) {
      const int G = ch.wlen[w];
      for (int r = 0; r < ch.wrounds[w]; ++r) {
        for (int s = 0; s < G; ++s, wd += 32) {
          for (int l = 0; l < 32; ++l) {
            const uint32_t d = wd[l];
            const int32_t xs = (int32_t)(d & 0xfff), ysl = (int32_t)((d >> 12) & 0xfff);
            if (d >> 24) return fail_("descriptor with flag bits");
            if (xs >= ch.nx) {
              if (xs >= ch.nx + 8) return fail_("descriptor reads beyond the zero X blocks");
              if (ysl != (l & 7)) return fail_("padding step does not read its class's zero block");
              continue;
            }
            if (xof[(size_t)xs] < 0) return fail_("descriptor reads an unstaged X slot");
            if (ysl >= ch.nyslots || yof[(size_t)ysl] < 0) return fail_("descriptor reads an unstaged Y slot");
            if ((ysl & 7) != (l & 7)) return fail_("lane reads a Y slot of another class");
            const int32_t yrow = (int32_t)(yof[(size_t)ysl] >> 20), q = (int32_t)(yof[(size_t)ysl] & 0xfffff);
            if (rb.xcol[(size_t)xof[(size_t)xs]] != yrow) return fail_("X block multiplied with the wrong Y row");
            lane_pending[(size_t)w * 32 + l].push_back(key(xof[(size_t)xs], yrow, q));
          }
          if (stats)
            for (int qd = 0; qd < 4; ++qd) {
              int degx = 1, degy = 1;
              for (int a = 0; a < 8; ++a) {
                const uint32_t da = wd[qd * 8 + a];
                int cx = 1, cy = 1;
                for (int b = 0; b < a; ++b) {
                  const uint32_t db = wd[qd * 8 + b];
                  const int32_t xa = da & 0xfff, xb = db & 0xfff, ya = (da >> 12) & 0xfff, yb = (db >> 12) & 0xfff;
                  bool dup = false;
                  for (int c2 = 0; c2 < b; ++c2) dup = dup || (int32_t)(wd[qd * 8 + c2] & 0xfff) == xb;
                  if (!dup && xa != xb && ((xa * xc16) & 7) == ((xb * xc16) & 7)) ++cx;
                  if (ya != yb && ((ya * yc16) & 7) == ((yb * yc16) & 7)) ++cy;
                }
                degx = std::max(degx, cx); degy = std::max(degy, cy);
              }
              stats->xq_clk += degx; stats->yq_clk += degy;
            }
        }
        if (!persist) {
          for (int l = 0; l < 32; ++l) {
            const uint32_t sw = wd[l];
            if (sw == PROG_NONE) continue;
            if ((int32_t)sw >= nslots) return fail_("store to a slot outside the staging area");
            if (slot_written[sw]) return fail_("staging slot written twice");
            slot_written[sw] = 1;
            auto& pend = lane_pending[(size_t)w * 32 + l];
            if (pend.empty()) return fail_("empty store");
            slot_prods[sw] = pend;
            pend.clear();
          }
          wd += 32;
        }
      }
    }
  }
  for (int t = 0; t < PROG_NT; ++t) {
    auto& pend = lane_pending[(size_t)t];
    if (persist) {
      const uint32_t sw = pstore[t];
      if (sw == PROG_NONE) { if (!pend.empty()) return fail_("lane with products has no staging slot"); continue; }
      if ((int32_t)sw >= nslots || slot_written[sw]) return fail_("bad final staging slot");
      slot_written[sw] = 1;
      slot_prods[sw] = pend;
    } else if (!pend.empty()) {
      return fail_("products after the last store of a lane");
    }
  }
  // overflow parts joined into their output block
  std::vector<char> ovf_used((size_t)p.novf, 0);
  for (int32_t f = 0; f < p.nfix; ++f) {
    const int32_t main = (int32_t)(fix[2 * f] & 0xffff), first = (int32_t)(fix[2 * f] >> 16), cnt = (int32_t)fix[2 * f + 1];
    if (main >= p.ncs || first < p.ncs || first + cnt > nslots) return fail_("fix entry out of range");
    for (int32_t k = 0; k < cnt; ++k) {
      if (ovf_used[(size_t)(first + k - p.ncs)]) return fail_("overflow slot joined twice");
      ovf_used[(size_t)(first + k - p.ncs)] = 1;
      if (!slot_written[(size_t)first + k]) return fail_("joined overflow slot never written");
      auto& g = slot_prods[(size_t)main];
      g.insert(g.end(), slot_prods[(size_t)first + k].begin(), slot_prods[(size_t)first + k].end());
    }
  }
  for (int32_t k = 0; k < p.novf; ++k) if (!ovf_used[(size_t)k]) return fail_("overflow slot never joined");
  // output rows as staged: crow must match the brick's C rows
  int32_t cs = 0;
  for (int32_t r = 0; r < nrows; ++r) {
    if ((int32_t)(crow[r] & 0xffff) != cs || (int32_t)(crow[r] >> 16) != rb.clen[r]) return fail_("staged output rows do not match C");
    cs += rb.clen[r];
  }
  if (cs != p.ncs || cs != (int32_t)items.size()) return fail_("staged output count");
  for (size_t s = 0; s < items.size(); ++s) {
    std::vector<uint64_t> want;
    for (const Prod& pr : items[s].prods) want.push_back(key(pr.x, pr.yrow, pr.q));
    std::sort(want.begin(), want.end());
    auto& g = slot_prods[s];   // items are in output order: item s <-> main slot s
    std::sort(g.begin(), g.end());
    if (want != g) return fail_("an output block does not receive exactly its block products");
  }
  if (stats) { stats->products += p.products; stats->lane_steps += p.lane_steps; }
  return true;
}

// ------------------------------------------------------------------ stage plans
namespace {

struct Cache {
  std::mutex mu;
  std::unordered_map<uint64_t, std::vector<std::pair<RelBrick, std::shared_ptr<Program>>>> map;
};

std::shared_ptr<Program> cached_build(Cache& cache, const ProgShape& sh, bool persist, int64_t budget, int round_len,
                                      RelBrick&& rb) {
  const uint64_t h = rb.hash();
  {
    std::lock_guard<std::mutex> g(cache.mu);
    auto it = cache.map.find(h);
    if (it != cache.map.end())
      for (auto& e : it->second)
        if (e.first == rb) return e.second;
  }
  auto p = std::make_shared<Program>();
  prog_build(sh, persist, budget, round_len, rb, *p);
  std::lock_guard<std::mutex> g(cache.mu);
  auto& bucket = cache.map[h];
  for (auto& e : bucket)
    if (e.first == rb) return e.second;
  bucket.emplace_back(std::move(rb), p);
  return p;
}

struct PlacedBrick {
  std::shared_ptr<Program> prog;
  std::vector<int32_t> inst;   // xsrc[nrows], outbase[nrows], ysrc[nyrows]
};

// relative structure + instance of the brick made of `rows` (rows of X)
void make_brick(const std::vector<int32_t>& rows, const int32_t* rowptr_x, const int32_t* colidx_x,
                const int32_t* rowptr_y, const int32_t* colidx_y, const int32_t* rowptr_c, const int32_t* colidx_c,
                RelBrick& rb, std::vector<int32_t>& inst) {
  std::vector<int32_t> ys, cols;
  for (int32_t i : rows) ys.insert(ys.end(), colidx_x + rowptr_x[i], colidx_x + rowptr_x[i + 1]);
  std::sort(ys.begin(), ys.end());
  ys.erase(std::unique(ys.begin(), ys.end()), ys.end());
  for (int32_t j : ys) cols.insert(cols.end(), colidx_y + rowptr_y[j], colidx_y + rowptr_y[j + 1]);
  std::sort(cols.begin(), cols.end());
  cols.erase(std::unique(cols.begin(), cols.end()), cols.end());
  rb = RelBrick();
  rb.ncols = (int32_t)cols.size();
  inst.clear();
  for (int32_t i : rows) inst.push_back(rowptr_x[i]);
  for (int32_t i : rows) inst.push_back(rowptr_c[i]);
  for (int32_t j : ys) inst.push_back(rowptr_y[j]);
  for (int32_t i : rows) {
    rb.xlen.push_back(rowptr_x[i + 1] - rowptr_x[i]);
    for (int32_t k = rowptr_x[i]; k < rowptr_x[i + 1]; ++k)
      rb.xcol.push_back((int32_t)(std::lower_bound(ys.begin(), ys.end(), colidx_x[k]) - ys.begin()));
    rb.clen.push_back(rowptr_c[i + 1] - rowptr_c[i]);
    for (int32_t k = rowptr_c[i]; k < rowptr_c[i + 1]; ++k)
      rb.ccol.push_back((int32_t)(std::lower_bound(cols.begin(), cols.end(), colidx_c[k]) - cols.begin()));
  }
  for (int32_t j : ys) {
    rb.ylen.push_back(rowptr_y[j + 1] - rowptr_y[j]);
    for (int32_t k = rowptr_y[j]; k < rowptr_y[j + 1]; ++k)
      rb.ycol.push_back((int32_t)(std::lower_bound(cols.begin(), cols.end(), colidx_y[k]) - cols.begin()));
  }
}

// serialises one program into the device blob format (ptap_prog.h); returns the word offset of its first chunk
int64_t serialise(bool persist, const Program& p, std::vector<uint32_t>& blob) {
  const size_t nch = p.chunks.size();
  std::vector<int64_t> start(nch), words(nch);
  int64_t at = (int64_t)blob.size();
  for (size_t c = 0; c < nch; ++c) {
    start[c] = at;
    words[c] = prog_blob_words(persist, c + 1 == nch, p.nrows, p.nfix, p.chunks[c]);
    at += words[c];
  }
  for (size_t c = 0; c < nch; ++c) {
    const ProgChunk& ch = p.chunks[c];
    const size_t b0 = blob.size();
    uint32_t h[PROG_H_WORDS] = {0};
    h[PROG_H_NX] = (uint32_t)ch.nx; h[PROG_H_NYSLOTS] = (uint32_t)ch.nyslots;
    h[PROG_H_NXRUN] = (uint32_t)ch.nxrun; h[PROG_H_NYCOPY] = (uint32_t)ch.nycopy;
    h[PROG_H_ROUNDS01] = (uint32_t)(uint16_t)ch.wrounds[0] | ((uint32_t)(uint16_t)ch.wrounds[1] << 16);
    h[PROG_H_ROUNDS23] = (uint32_t)(uint16_t)ch.wrounds[2] | ((uint32_t)(uint16_t)ch.wrounds[3] << 16);
    h[PROG_H_LEN01] = (uint32_t)(uint16_t)ch.wlen[0] | ((uint32_t)(uint16_t)ch.wlen[1] << 16);
    h[PROG_H_LEN23] = (uint32_t)(uint16_t)ch.wlen[2] | ((uint32_t)(uint16_t)ch.wlen[3] << 16);
    h[PROG_H_PROG_WORDS] = (uint32_t)ch.blob_words;
    h[PROG_H_NCS] = (uint32_t)p.ncs; h[PROG_H_NOVF] = (uint32_t)p.novf; h[PROG_H_NFIX] = (uint32_t)p.nfix;
    h[PROG_H_NEXT_BLOB] = c + 1 < nch ? (uint32_t)start[c + 1] : 0xffffffffu;
    h[PROG_H_NEXT_WORDS] = c + 1 < nch ? (uint32_t)words[c + 1] : 0u;
    blob.insert(blob.end(), h, h + PROG_H_WORDS);
    for (int32_t e = ch.xrun0; e < ch.xrun0 + ch.nxrun; ++e) {
      const XRun& xr = p.xruns[(size_t)e];
      blob.push_back((uint32_t)xr.row | ((uint32_t)xr.k0 << 16));
      blob.push_back((uint32_t)xr.n | ((uint32_t)xr.dst << 16));
    }
    for (int32_t e = ch.ycopy0; e < ch.ycopy0 + ch.nycopy; ++e) {
      const YCopy& yc = p.ycopies[(size_t)e];
      blob.push_back((uint32_t)yc.yrow | ((uint32_t)yc.q << 12) | ((uint32_t)yc.slot << 20));
    }
    while ((blob.size() - b0) & 3) blob.push_back(0);
    blob.insert(blob.end(), p.blob.begin() + ch.blob0, p.blob.begin() + ch.blob0 + ch.blob_words);
    if (c + 1 == nch) blob.insert(blob.end(), p.tabs.begin(), p.tabs.end());
    while ((blob.size() - b0) & 3) blob.push_back(0);
    if ((int64_t)(blob.size() - b0) != words[c]) return -1;
  }
  return start[0];
}

void flatten(const ProgShape& sh, bool persist, std::vector<PlacedBrick>& placed, Cache& cache, bool keep, ProgPlan& out) {
  out.ok = false; out.persist = persist; out.shape = sh;
  std::unordered_map<const Program*, int32_t> id;
  std::vector<int64_t> blob_at, blob_words;
  int64_t max_rec = 0, max_blob = 0, max_xy = 0, max_cs = 0;
  out.rec_off.push_back(0);
  for (PlacedBrick& pb : placed) {
    const Program& p = *pb.prog;
    if (!p.ok) { out.why = p.why; return; }
    auto it = id.find(pb.prog.get());
    int32_t pid;
    if (it == id.end()) {
      pid = (int32_t)blob_at.size();
      id.emplace(pb.prog.get(), pid);
      const int64_t at = serialise(persist, p, out.blob);
      if (at < 0 || out.blob.size() >= (size_t)1 << 31) { out.why = "plan too large"; return; }
      blob_at.push_back(at);
      blob_words.push_back(prog_blob_words(persist, p.chunks.size() == 1, p.nrows, p.nfix, p.chunks[0]));
      out.prog_uses.push_back(0);
      max_rec = std::max(max_rec, p.rec_bytes); max_blob = std::max(max_blob, p.blob_bytes);
      max_xy = std::max(max_xy, p.xy_bytes); max_cs = std::max(max_cs, p.smem_cs);
      out.nchunks += (int64_t)p.chunks.size();
      out.nycopies += (int64_t)p.ycopies.size();
    } else {
      pid = it->second;
    }
    out.prog_uses[(size_t)pid]++;
    const int32_t rw = prog_rec_words(p.nrows, p.nyrows);
    if ((int64_t)out.rec.size() + rw >= (1LL << 31)) { out.why = "plan too large"; return; }
    const size_t r0 = out.rec.size();
    out.rec.push_back((uint32_t)blob_at[(size_t)pid]);
    out.rec.push_back((uint32_t)blob_words[(size_t)pid]);
    out.rec.push_back((uint32_t)p.nrows);
    out.rec.push_back((uint32_t)p.nyrows);
    for (int32_t v : pb.inst) out.rec.push_back((uint32_t)v);
    out.rec.resize(r0 + (size_t)rw, 0u);
    out.rec_off.push_back((int32_t)out.rec.size());

    out.stats.products += p.products;
    out.stats.lane_steps += p.lane_steps;
  }
  out.nbricks = (int64_t)placed.size();
  out.nprograms = (int64_t)blob_at.size();
  out.rec_max_bytes = (int32_t)max_rec; out.blob_max_bytes = (int32_t)max_blob;
  out.max_smem = 3 * max_rec + 2 * max_blob + max_xy + max_cs;
  out.stats.bricks = out.nbricks;
  out.stats.programs = out.nprograms;
  out.stats.max_smem = out.max_smem;
  out.stats.plan_bytes = (int64_t)out.rec_off.size() * 4 + (int64_t)out.rec.size() * 4 + (int64_t)out.blob.size() * 4;
  if (keep)
    for (auto& kv : cache.map)
      for (auto& e : kv.second) {
        auto f = id.find(e.second.get());
        out.kept_id.push_back(f == id.end() ? -1 : f->second);
        out.kept.emplace_back(std::move(e.first), e.second);
      }
  out.ok = true;
}

}  // namespace

// Stage 1: fine rows that share a "home" coarse column are staged together: home(i) = the column of AP's row i that
// receives the most block products -- for an aggregation-based P the row's own aggregate, so a group's Y rows are the
// aggregate's neighbourhood.  Purely structural; it only decides scheduling.  A group whose program does not fit the
// shared-memory budget is halved (by row order) until it does.
static void plan_stage1_once(const ProgShape& sh, int64_t budget, int round_len, int32_t n, const int32_t* rowptr_a, const int32_t* colidx_a,
                      const int32_t* rowptr_p, const int32_t* colidx_p, int32_t nc, const int32_t* rowptr_ap,
                      const int32_t* colidx_ap, ProgPlan& out, bool keep) {
  out = ProgPlan();
  std::vector<int32_t> home((size_t)n, 0);
#pragma omp parallel
  {
    std::vector<int32_t> cnt((size_t)nc, 0);
#pragma omp for schedule(static)
    for (int32_t i = 0; i < n; ++i) {
      int32_t best = -1, bestn = 0;
      for (int32_t k = rowptr_a[i]; k < rowptr_a[i + 1]; ++k) {
        const int32_t j = colidx_a[k];
        for (int32_t q = rowptr_p[j]; q < rowptr_p[j + 1]; ++q) {
          const int32_t c = ++cnt[(size_t)colidx_p[q]];
          if (c > bestn || (c == bestn && colidx_p[q] < best)) { bestn = c; best = colidx_p[q]; }
        }
      }
      for (int32_t k = rowptr_a[i]; k < rowptr_a[i + 1]; ++k) {
        const int32_t j = colidx_a[k];
        for (int32_t q = rowptr_p[j]; q < rowptr_p[j + 1]; ++q) cnt[(size_t)colidx_p[q]] = 0;
      }
      home[i] = best < 0 ? 0 : best;
    }
  }
  std::vector<int32_t> gptr((size_t)nc + 2, 0), grows((size_t)n);
  for (int32_t i = 0; i < n; ++i) gptr[(size_t)home[i] + 1]++;
  for (int32_t j = 0; j < nc; ++j) gptr[(size_t)j + 1] += gptr[j];
  {
    std::vector<int32_t> fill(gptr.begin(), gptr.end() - 1);
    for (int32_t i = 0; i < n; ++i) grows[(size_t)fill[home[i]]++] = i;
  }
  Cache cache;
  std::vector<std::vector<PlacedBrick>> per((size_t)nc);
  const int xs = prog_xs(sh), yc = prog_yc16(sh);
#pragma omp parallel
  {
    std::vector<int32_t> rows, inst;
#pragma omp for schedule(dynamic, 16)
    for (int32_t J = 0; J < nc; ++J) {
      const int32_t g0 = gptr[J], n = gptr[(size_t)J + 1] - g0;
      if (n == 0) continue;
      // the group is cut into k bricks of consecutive rows, k = the cheapest (modelled cycles) of the first few that
      // fit the shared-memory budget: a brick a little smaller than the budget allows can fill its rounds better
      std::vector<PlacedBrick> best;
      int64_t best_cost = -1;
      int tried_fitting = 0;
      for (int32_t k = 1; k <= n && tried_fitting < 4; ++k) {
        std::vector<PlacedBrick> cand;
        int64_t cost = 0;
        bool ok = true;
        for (int32_t b = 0; b < k && ok; ++b) {
          const int32_t r0 = (int32_t)((int64_t)n * b / k), r1 = (int32_t)((int64_t)n * (b + 1) / k);
          rows.assign(grows.begin() + g0 + r0, grows.begin() + g0 + r1);
          RelBrick rb;
          make_brick(rows, rowptr_a, colidx_a, rowptr_p, colidx_p, rowptr_ap, colidx_ap, rb, inst);
          const int64_t lower = (int64_t)(rb.xcol.size() + 8) * xs * 8 + (int64_t)rb.ycol.size() * yc * 16 +
                                (int64_t)rb.ccol.size() * sh.M * sh.N * 8;
          std::shared_ptr<Program> p;
          if (lower <= budget) p = cached_build(cache, sh, false, budget, round_len, std::move(rb));
          if (!p || !p->ok) {
            ok = false;
            if (k == n) {   // single rows that do not fit: report through the plan
              if (!p) { p = std::make_shared<Program>(); p->why = "a row does not fit the shared-memory budget"; }
              cand.push_back(PlacedBrick{p, inst});
            }
            break;
          }
          cost += p->cost;
          cand.push_back(PlacedBrick{p, inst});
        }
        if (ok) {
          ++tried_fitting;
          if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = std::move(cand); }
        } else if (k == n && best_cost < 0) {
          best = std::move(cand);   // carries the failure
        }
      }
      per[(size_t)J] = std::move(best);
    }
  }
  std::vector<PlacedBrick> placed;
  for (auto& v : per)
    for (auto& pb : v) placed.push_back(std::move(pb));
  flatten(sh, false, placed, cache, keep, out);
}

// The CTA's shared memory is the largest staged part plus the largest output staging area of any brick, which can
// exceed the per-brick budget a little: the per-brick budget is lowered until the sum fits.
void prog_plan_stage1(const ProgShape& sh, int64_t budget, int round_len, int32_t n, const int32_t* rowptr_a, const int32_t* colidx_a,
                      const int32_t* rowptr_p, const int32_t* colidx_p, int32_t nc, const int32_t* rowptr_ap,
                      const int32_t* colidx_ap, ProgPlan& out, bool keep) {
  int64_t b = budget;
  for (int attempt = 0; attempt < 4; ++attempt) {
    plan_stage1_once(sh, b, round_len, n, rowptr_a, colidx_a, rowptr_p, colidx_p, nc, rowptr_ap, colidx_ap, out, keep);
    if (!out.ok || out.max_smem <= budget) return;
    b -= (out.max_smem - budget) + 512;
  }
  out.ok = false;
  out.why = "bricks do not fit the shared-memory budget";
}

static void plan_stage2_once(const ProgShape& sh, int64_t budget, int32_t nc, const int32_t* rowptr_r, const int32_t* colidx_r,
                      const int32_t* rowptr_ap, const int32_t* colidx_ap, const int32_t* rowptr_c,
                      const int32_t* colidx_c, ProgPlan& out, bool keep) {
  out = ProgPlan();
  Cache cache;
  std::vector<PlacedBrick> placed((size_t)nc);
#pragma omp parallel
  {
    std::vector<int32_t> rows(1), inst;
#pragma omp for schedule(dynamic, 16)
    for (int32_t I = 0; I < nc; ++I) {
      rows[0] = I;
      RelBrick rb;
      make_brick(rows, rowptr_r, colidx_r, rowptr_ap, colidx_ap, rowptr_c, colidx_c, rb, inst);
      placed[(size_t)I] = PlacedBrick{cached_build(cache, sh, true, budget, 0, std::move(rb)), inst};
    }
  }
  flatten(sh, true, placed, cache, keep, out);
}

// Stage 2: one brick per coarse row I; its R row is cut into chunks that fit the budget.
void prog_plan_stage2(const ProgShape& sh, int64_t budget, int32_t nc, const int32_t* rowptr_r, const int32_t* colidx_r,
                      const int32_t* rowptr_ap, const int32_t* colidx_ap, const int32_t* rowptr_c,
                      const int32_t* colidx_c, ProgPlan& out, bool keep) {
  int64_t b = budget;
  for (int attempt = 0; attempt < 4; ++attempt) {
    plan_stage2_once(sh, b, nc, rowptr_r, colidx_r, rowptr_ap, colidx_ap, rowptr_c, colidx_c, out, keep);
    if (!out.ok || out.max_smem <= budget) return;
    b -= (out.max_smem - budget) + 512;
  }
  out.ok = false;
  out.why = "bricks do not fit the shared-memory budget";
}

}  // namespace bsramg
