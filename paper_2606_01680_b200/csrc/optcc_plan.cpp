// Host planner of liboptcc: builds the ell-weighted stage / chunk / step plan of OPTCC.
//
// Written from docs/PLAN_SPEC.md (which freezes the canonical reading of PAPER.md 4.1-4.4, App. C/D/E) and the
// paper itself; citations are PAPER.md:<line>.  Pure host C++, no CUDA: closed-form rules, O(p k) flows
// ("closed-form rules ... O(pk)").  Compiled with -ffp-contract=off: the one floating-point
// quantity that decides integers (the P2P share, PLAN_SPEC 2) must round exactly as the spec says.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <mutex>
#include <thread>
#include <new>

#include "optcc_internal.h"

// ---- raw table memory with a small process-wide cache (optcc_internal.h) ----
namespace {
struct RawBlock { void* p; size_t bytes; };
std::mutex g_raw_mutex;
std::vector<RawBlock> g_raw_cache;                 // at most RAW_CACHE_BLOCKS freed blocks
constexpr size_t RAW_CACHE_BLOCKS = 12;
constexpr size_t RAW_CACHE_MIN = size_t(1) << 16;  // smaller blocks go straight to malloc / free
constexpr size_t RAW_CACHE_MAX = size_t(1) << 30;  // total bytes kept
}  // namespace

void* optcc_raw_alloc(size_t bytes) {
  if (bytes == 0) bytes = 64;
  if (bytes >= RAW_CACHE_MIN) {
    std::lock_guard<std::mutex> lock(g_raw_mutex);
    size_t best = SIZE_MAX;
    for (size_t i = 0; i < g_raw_cache.size(); ++i)   // smallest cached block that fits without wasting more than half
      if (g_raw_cache[i].bytes >= bytes && g_raw_cache[i].bytes <= 2 * bytes &&
          (best == SIZE_MAX || g_raw_cache[i].bytes < g_raw_cache[best].bytes)) best = i;
    if (best != SIZE_MAX) {
      void* p = g_raw_cache[best].p;
      g_raw_cache.erase(g_raw_cache.begin() + best);
      return p;
    }
  }
  return std::aligned_alloc(64, (bytes + 63) & ~size_t(63));
}

// (the block's true capacity is not tracked: a recycled block is handed out again by the size it was freed with, which
//  is the size its last owner asked for -- never more than what was allocated)
void optcc_raw_free(void* p, size_t bytes) {
  if (!p) return;
  if (bytes >= RAW_CACHE_MIN) {
    std::lock_guard<std::mutex> lock(g_raw_mutex);
    // the newest block stays, the oldest ones go: a job that moves on to another plan shape must find ITS blocks cached
    if (bytes <= RAW_CACHE_MAX) {
      g_raw_cache.push_back(RawBlock{p, bytes});
      size_t total = 0;
      for (const auto& b : g_raw_cache) total += b.bytes;
      while (g_raw_cache.size() > RAW_CACHE_BLOCKS || total > RAW_CACHE_MAX) {
        total -= g_raw_cache.front().bytes;
        std::free(g_raw_cache.front().p);
        g_raw_cache.erase(g_raw_cache.begin());
      }
      return;
    }
  }
  std::free(p);
}

namespace {

// x mod H for -H <= x < 2H (all the rules need: ring positions shifted by at most one lap)
inline uint32_t modH(int64_t x, int64_t H) { return (uint32_t)(x < 0 ? x + H : (x >= H ? x - H : x)); }

// Everything the closed-form rules of PLAN_SPEC 4 need, fixed before the first flow is written.  The table is never
// sorted: emit_step() lists the flows of one step directly in PLAN_SPEC 3 order (link, stage, src, dst, off), so the
// steps can be counted and filled independently ("closed-form rules ... O(pk)").
struct Geom {
  uint32_t p = 0, g = 1, q = 0, m = 0, H = 0, k = 0, nsec = 0;
  uint32_t construction = 0, ordering = 2;
  uint32_t P = 0;        // windows per body: H (C1, C3 with one straggler server), H + m - 1 otherwise (:788)
  uint32_t D = 0;        // C3: the NIC body of segment b is body b + D
  uint32_t n_steps = 0;
  bool bubbles = false;
  const uint32_t* healthy = nullptr;      // server indices, ascending
  const uint32_t* stragglers = nullptr;   // server indices, PLAN_SPEC 1 order (ell descending)
  std::vector<uint32_t> str_by_rank;      // positions in `stragglers`, by server index ascending (S3: src order)
  // regions: the sections in (part, segment, section) order, then the P2P pieces; UINT32_MAX = empty interval (dropped)
  std::vector<uint32_t> sec_reg, p2p_reg;
  const uint64_t* region_off = nullptr;
  const uint64_t* region_len = nullptr;
  uint32_t sec(uint32_t lam, uint32_t b, uint32_t c) const { return sec_reg[(size_t(lam) * k + b) * nsec + c]; }
};

// One flow of step t; region == UINT32_MAX: a zero-length range (PLAN_SPEC 2: dropped).
struct CountSink {
  static constexpr bool kOrdered = false;   // the order inside a step does not matter for counting
  uint32_t n = 0;
  void operator()(uint32_t, uint8_t, uint8_t, uint8_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t region) {
    n += region != UINT32_MAX;
  }
};
struct CountAllSink {   // no region is empty: every rule application is a flow (the arguments are never computed)
  static constexpr bool kOrdered = false;
  uint32_t n = 0;
  void operator()(uint32_t, uint8_t, uint8_t, uint8_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t) { ++n; }
};
struct FillSink {
  static constexpr bool kOrdered = true;
  const Geom* G;
  uint32_t* region_count = nullptr;   // this chunk's flows per region
  optcc_flow_t* out;        // next record
  uint32_t* out_region;
  uint64_t reduce_elems = 0, copy_elems = 0;
  void operator()(uint32_t step, uint8_t op, uint8_t stage, uint8_t link, uint32_t part, uint32_t src, uint32_t dst,
                  uint32_t seg, uint32_t sec, uint32_t region) {
    if (region == UINT32_MAX) return;
    optcc_flow_t f;
    f.off = G->region_off[region]; f.len = G->region_len[region];
    f.step = step; f.seg = seg; f.sec = sec;
    f.src = (uint16_t)src; f.dst = (uint16_t)dst; f.op = op; f.stage = stage; f.link = link; f.part = (uint8_t)part;
    f.reserved = 0;
    *out++ = f;
    *out_region++ = region;
    region_count[region]++;
    (op == OPTCC_OP_REDUCE ? reduce_elems : copy_elems) += f.len;
  }
};

// The flows of step t in table order (PLAN_SPEC 3: link, stage, src, dst, off).  Within one stage the senders are
// visited in increasing rank, and a sender has one flow per stage and step except on the NVLink rings (see below).
template <class Sink>
void emit_step(const Geom& G, uint32_t t, Sink& out) {
  const uint32_t H = G.H, k = G.k, g = G.g, m = G.m;
  if (G.construction == OPTCC_C0) {
    // plain ring: reduce-scatter p-1 hops then all-gather p-1 hops (:52, :72)
    const uint32_t p = G.p;
    if (t < p - 1) {
      for (uint32_t j = 0; j < p; ++j)
        out(t, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, 0, j, (j + 1 == p ? 0 : j + 1), 0, modH(int64_t(j) - t, p), G.sec(0, 0, modH(int64_t(j) - t, p)));
    } else {
      const uint32_t tt = t - (p - 1);
      for (uint32_t j = 0; j < p; ++j)
        out(t, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, 0, j, (j + 1 == p ? 0 : j + 1), 0, modH(int64_t(j) + 1 - tt, p), G.sec(0, 0, modH(int64_t(j) + 1 - tt, p)));
    }
    return;
  }
  if (G.construction == OPTCC_C1 && G.ordering == 3) {
    // C1'': the four-pattern mix of :144-155 (PLAN_SPEC 4 C1'').  Segment b = 4 gamma + pattern; patterns A, C (0, 2) use
    // ordering (1) S1 -> S2 -> S3 -> S4, patterns B, D (1, 3) ordering (2) S3 -> S1 -> S4 -> S2, one stage per body; A and
    // B start in body 4 gamma, C and D one body later.  seg_at: the segment of `pattern` whose stage number `idx` (in
    // its own ordering) falls into this body, or none.
    const uint32_t beta = t / H, w = t % H, sg = G.stragglers[0];
    const uint32_t a = w, d = (w + 1) % H;
    auto seg_at = [&](uint32_t pattern, uint32_t idx, uint32_t* b) {
      const uint32_t shift = (pattern >= 2 ? 1u : 0u) + idx;
      if (beta < shift || (beta - shift) % 4 != 0) return false;
      *b = beta - shift + pattern;
      return *b < k;
    };
    uint32_t b;
    // Stage 1: A, C in their first body, B, D in their second; ring link j idle in window j (ascending b = ascending offset)
    for (uint32_t j = 0; j < H; ++j) {
      if (w == j) continue;
      const uint32_t hop = w < j ? w : w - 1, c = modH(int64_t(j) - hop, H);
      for (uint32_t pat = 0; pat < 4; ++pat)
        if (seg_at(pat, pat & 1u ? 1 : 0, &b))
          out(t, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, 0, G.healthy[j], G.healthy[j + 1 == H ? 0 : j + 1], b, c, G.sec(0, b, c));
    }
    // Stage 2: A, C (second body) the straggler adds its own data to the uploaded partial sum (:130-132);
    //          B, D (fourth body) the owner sends the global sum to the straggler (:138 ordering (2))
    for (uint32_t pat = 0; pat < 4; ++pat)
      if (seg_at(pat, pat & 1u ? 3 : 1, &b))
        out(t, pat & 1u ? OPTCC_OP_COPY : OPTCC_OP_REDUCE, OPTCC_S2, OPTCC_LINK_NIC, 0, G.healthy[a], sg, b, (a + 1) % H, G.sec(0, b, (a + 1) % H));
    // Stage 3: A, C (third body) the global sum returns to the uploader's ring successor (:132, R11);
    //          B, D (first body) the straggler's raw section is folded in at its owner (:138)
    for (uint32_t pat = 0; pat < 4; ++pat)
      if (seg_at(pat, pat & 1u ? 0 : 2, &b)) {
        if (pat & 1u) out(t, OPTCC_OP_REDUCE, OPTCC_S3, OPTCC_LINK_NIC, 0, sg, G.healthy[d], b, (d + 1) % H, G.sec(0, b, (d + 1) % H));
        else out(t, OPTCC_OP_COPY, OPTCC_S3, OPTCC_LINK_NIC, 0, sg, G.healthy[d], b, d, G.sec(0, b, d));
      }
    // Stage 4: A, C in their fourth body (the all-gather of section c starts at healthy c), B, D in their third
    for (uint32_t j = 0; j < H; ++j) {
      if (w == j) continue;
      const uint32_t hop = w < j ? w : w - 1;
      for (uint32_t pat = 0; pat < 4; ++pat)
        if (seg_at(pat, pat & 1u ? 2 : 3, &b)) {
          const uint32_t c = pat & 1u ? modH(int64_t(j) + 1 - hop, H) : modH(int64_t(j) - hop, H);
          out(t, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, 0, G.healthy[j], G.healthy[j + 1 == H ? 0 : j + 1], b, c, G.sec(0, b, c));
        }
    }
    if (G.bubbles && beta < k)
      out(t, OPTCC_OP_REDUCE, OPTCC_BUB_UP, OPTCC_LINK_NIC, 0, G.healthy[a], sg, beta, 0, G.p2p_reg[beta]);
    if (G.bubbles && beta >= 1)
      out(t, OPTCC_OP_COPY, OPTCC_BUB_DOWN, OPTCC_LINK_NIC, 0, sg, G.healthy[d], beta - 1, 0, G.p2p_reg[beta - 1]);
    return;
  }
  if (G.construction == OPTCC_C1 && G.ordering == 1) {
    // C1': ordering (1) of :138, S1 -> S2 -> S3 -> S4, one stage per body (PLAN_SPEC 4 C1')
    const uint32_t Bd = t / H, w = t % H, sg = G.stragglers[0];
    const uint32_t a = w, d = (w + 1) % H;
    if (Bd < k)       // Stage 1: partial sums of the healthy servers (:126); ring link j idle in window j
      for (uint32_t j = 0; j < H; ++j) {
        if (w == j) continue;
        const uint32_t hop = w < j ? w : w - 1, c = modH(int64_t(j) - hop, H);
        out(t, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, 0, G.healthy[j], G.healthy[j + 1 == H ? 0 : j + 1], Bd, c, G.sec(0, Bd, c));
      }
    if (Bd >= 1 && Bd <= k)       // Stage 2: the straggler adds its own data to the uploaded partial sum (:130-132)
      out(t, OPTCC_OP_REDUCE, OPTCC_S2, OPTCC_LINK_NIC, 0, G.healthy[a], sg, Bd - 1, (a + 1) % H, G.sec(0, Bd - 1, (a + 1) % H));
    if (Bd >= 2 && Bd <= k + 1)   // Stage 3: the global sum returns to the uploader's ring successor (:132, R11)
      out(t, OPTCC_OP_COPY, OPTCC_S3, OPTCC_LINK_NIC, 0, sg, G.healthy[d], Bd - 2, d, G.sec(0, Bd - 2, d));
    if (Bd >= 3)      // Stage 4: the all-gather of section c starts at healthy c (:136)
      for (uint32_t j = 0; j < H; ++j) {
        if (w == j) continue;
        const uint32_t hop = w < j ? w : w - 1, c = modH(int64_t(j) - hop, H);
        out(t, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, 0, G.healthy[j], G.healthy[j + 1 == H ? 0 : j + 1], Bd - 3, c, G.sec(0, Bd - 3, c));
      }
    if (G.bubbles && Bd < k)
      out(t, OPTCC_OP_REDUCE, OPTCC_BUB_UP, OPTCC_LINK_NIC, 0, G.healthy[a], sg, Bd, 0, G.p2p_reg[Bd]);
    if (G.bubbles && Bd >= 1 && Bd <= k)
      out(t, OPTCC_OP_COPY, OPTCC_BUB_DOWN, OPTCC_LINK_NIC, 0, sg, G.healthy[d], Bd - 1, 0, G.p2p_reg[Bd - 1]);
    return;
  }
  // C1 / C2 / C3: NIC flows of body BB = Bd + D, window w (leaders: local GPU lam of every server, :854)
  const uint32_t P = G.P, D = G.D, BB = t / P, w = t % P;
  if (BB >= D && BB - D <= k) {
    const uint32_t Bd = BB - D;
    // ring link j (healthy j -> j+1) is idle in windows [j, j+m); hop `hop` sits in window W(j, hop)
    if (Bd < k)   // Stage 1, segment Bd: add own section and forward (:126)
      for (uint32_t j = 0; j < H; ++j) {
        if (w >= j && w < j + m) continue;
        const uint32_t hop = w < j ? w : w - m, c = modH(int64_t(j) - hop, H);
        for (uint32_t lam = 0; lam < g; ++lam)
          out(t, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, lam, G.healthy[j] * g + lam, G.healthy[j + 1 == H ? 0 : j + 1] * g + lam, Bd, c, G.sec(lam, Bd, c));
      }
    // straggler i is active in windows [i, i+H) with uploader a = w - i, downloader d = (a+1) mod H
    if (Bd >= 1) {  // Stage 2: the owner uploads the complete sum to the straggler (:130; ordering (2) :138); by sender a
      const uint32_t i_hi = std::min<uint32_t>(m - 1, w);
      for (uint32_t i = i_hi + 1; i-- > 0;) {
        const uint32_t a = w - i;
        if (a >= H) break;
        for (uint32_t lam = 0; lam < g; ++lam)
          out(t, OPTCC_OP_COPY, OPTCC_S2, OPTCC_LINK_NIC, lam, G.healthy[a] * g + lam, G.stragglers[i] * g + lam, Bd - 1, (a + 1) % H, G.sec(lam, Bd - 1, (a + 1) % H));
      }
    }
    if (Bd < k)     // Stage 3: the straggler's raw section is folded in at its owner (:132, :138); by sender (straggler rank)
      for (uint32_t ii = 0; ii < m; ++ii) {
        const uint32_t i = G.str_by_rank[ii];
        if (w < i || w - i >= H) continue;
        const uint32_t a = w - i, d = (a + 1) % H;
        for (uint32_t lam = 0; lam < g; ++lam)
          out(t, OPTCC_OP_REDUCE, OPTCC_S3, OPTCC_LINK_NIC, lam, G.stragglers[i] * g + lam, G.healthy[d] * g + lam, Bd, (d + 1) % H, G.sec(lam, Bd, (d + 1) % H));
      }
    if (Bd >= 1)    // Stage 4, segment Bd-1: forward the complete sum (:136)
      for (uint32_t j = 0; j < H; ++j) {
        if (w >= j && w < j + m) continue;
        const uint32_t hop = w < j ? w : w - m, c = modH(int64_t(j) + 1 - hop, H);
        for (uint32_t lam = 0; lam < g; ++lam)
          out(t, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, lam, G.healthy[j] * g + lam, G.healthy[j + 1 == H ? 0 : j + 1] * g + lam, Bd - 1, c, G.sec(lam, Bd - 1, c));
      }
    if (G.bubbles) {   // (one straggler, g = 1, P = H)
      const uint32_t a = w, d = (w + 1) % H, sg = G.stragglers[0];
      if (Bd < k)    // bubble-up: healthy a's raw P2P piece into the straggler (:165, R9)
        out(t, OPTCC_OP_REDUCE, OPTCC_BUB_UP, OPTCC_LINK_NIC, 0, G.healthy[a], sg, Bd, 0, G.p2p_reg[Bd]);
      if (Bd >= 1)   // bubble-down: the straggler returns the P2P result (:165)
        out(t, OPTCC_OP_COPY, OPTCC_BUB_DOWN, OPTCC_LINK_NIC, 0, sg, G.healthy[d], Bd - 1, 0, G.p2p_reg[Bd - 1]);
    }
  }
  if (G.construction != OPTCC_C3) return;
  // NVLink rings of every server (link 1 sorts after the NIC flows).  Hop h of (part lam, segment b, section c) sits at
  // step b P + c + h (collect) resp. (b + D + 2) P + c + h (distribute); a GPU can send several flows of one stage in
  // one step (one per h, each for another part), all to the same neighbour: those are ordered by offset, i.e. by
  // (lam, b, c) since the parts are consecutive ranges.
  struct Cand { uint32_t lam, b, c; };
  Cand cand[256];
  auto nv_stage = [&](bool collect) {
    const uint64_t shift = collect ? 0 : uint64_t(D + 2) * P;
    if (t < shift) return;
    const uint64_t tt = t - shift;
    for (uint32_t v = 0; v < G.q; ++v)
      for (uint32_t x = 0; x < g; ++x) {     // sender: local GPU x of server v
        uint32_t nc = 0;
        uint32_t b = uint32_t(tt / P), c = uint32_t(tt % P);          // (b, c) of hop h: b P + c = tt - h
        for (uint32_t h = 0; h + 1 < g && h <= tt; ++h) {
          if (h) { if (c == 0) { c = P - 1; --b; } else --c; }
          if (b >= k || c >= H) continue;
          // collect: local (lam-1-h) -> (lam-2-h) (backward ring, the leader only receives, :862, :875, :894);
          // distribute: local (lam+h) -> (lam+h+1) (forward ring, the leader sends first, :863, :876, :894)
          uint32_t lam;
          if (collect) { lam = x + 1 + h; if (lam >= g) lam -= g; }      // (h <= g-2, x <= g-1: at most one lap)
          else lam = x >= h ? x - h : x + g - h;
          Cand cd{lam, b, c};
          uint32_t pos = nc++;
          if (Sink::kOrdered)
            while (pos > 0 && (cand[pos - 1].lam > cd.lam || (cand[pos - 1].lam == cd.lam &&
                   (cand[pos - 1].b > cd.b || (cand[pos - 1].b == cd.b && cand[pos - 1].c > cd.c))))) {
              cand[pos] = cand[pos - 1];
              --pos;
            }
          cand[pos] = cd;
        }
        const uint32_t src = v * g + x, dst = v * g + (collect ? (x + g - 1) % g : (x + 1) % g);
        for (uint32_t i = 0; i < nc; ++i)
          out(t, collect ? OPTCC_OP_REDUCE : OPTCC_OP_COPY, collect ? OPTCC_N_COLLECT : OPTCC_N_DISTRIBUTE, OPTCC_LINK_NVLINK,
              cand[i].lam, src, dst, cand[i].b, cand[i].c, G.sec(cand[i].lam, cand[i].b, cand[i].c));
      }
  };
  nv_stage(true);
  nv_stage(false);
}

// Storage kinds for bf16 plans: walk the table once with the number of contributors every
// (rank, region) holds.  A region holding 1 or all p contributors lives in the rank buffer (bf16); a partial
// sum (1 < count < p) lives in the fp32 shadow.  All flows of one step read the state before the step.
}  // namespace

void optcc_assign_kinds(optcc_plan_t* pl) {
  const uint32_t p = pl->info.p;
  const size_t nf = pl->flows.size();
  if (pl->info.dtype != OPTCC_BF16) return;      // f32 plans: the three arrays stay empty (everything is OPTCC_KIND_BUF)
  pl->kind_src.assign(nf, OPTCC_KIND_BUF);
  pl->kind_dst_in.assign(nf, OPTCC_KIND_BUF);
  pl->kind_dst_out.assign(nf, OPTCC_KIND_BUF);
  const size_t nr = pl->region_offs.size();
  std::vector<uint16_t> cnt(size_t(p) * nr, 1);
  auto region = [&](uint32_t i) { return size_t(pl->flow_region[i]); };
  auto kind_of = [&](uint16_t c) -> uint8_t { return (c == 1 || c >= p) ? OPTCC_KIND_BUF : OPTCC_KIND_F32; };
  std::vector<uint16_t> src_cnt;
  for (uint32_t t = 0; t < pl->info.n_steps; ++t) {
    uint32_t lo = pl->step_begin[t], hi = pl->step_begin[t + 1];
    src_cnt.resize(hi - lo);
    for (uint32_t i = lo; i < hi; ++i) src_cnt[i - lo] = cnt[size_t(pl->flows[i].src) * nr + region(i)];
    for (uint32_t i = lo; i < hi; ++i) {
      const optcc_flow_t& f = pl->flows[i];
      uint16_t& cd = cnt[size_t(f.dst) * nr + region(i)];
      uint16_t cs = src_cnt[i - lo];
      pl->kind_src[i] = kind_of(cs);
      pl->kind_dst_in[i] = kind_of(cd);
      uint16_t out = (f.op == OPTCC_OP_REDUCE) ? uint16_t(cs + cd) : cs;
      pl->kind_dst_out[i] = kind_of(out);
      cd = out;
    }
  }
}

extern "C" int optcc_plan_ex(int p, int g, const double* ell, uint64_t n, int dtype, const optcc_opts_t* opts,
                             optcc_plan_t** out) {
  auto t_begin = std::chrono::steady_clock::now();
  if (!out || !ell) return OPTCC_EINVAL;
  // ---- PLAN_SPEC 1: validation and classification (PAPER.md:68 "p >= 3", :78, :274, :850) ----
  if (p < 3 || p > 65535 || g < 1 || p % g != 0) return OPTCC_EINVAL;
  const uint32_t schedule = opts ? opts->schedule : OPTCC_SCHED_OPTCC;
  if (schedule != OPTCC_SCHED_OPTCC && schedule != OPTCC_SCHED_RING_DEGRADED) return OPTCC_EINVAL;
  if (schedule == OPTCC_SCHED_RING_DEGRADED && g != 1) return OPTCC_EUNSUPPORTED;   // PLAN_SPEC 1: ring baseline, g = 1
  for (int i = 0; i < p; ++i)
    if (!std::isfinite(ell[i]) || ell[i] < 1.0) return OPTCC_EINVAL;
  const uint32_t q = uint32_t(p / g);
  for (uint32_t v = 0; v < q; ++v)
    for (int i = 1; i < g; ++i)
      if (ell[v * g + i] != ell[v * g]) return OPTCC_EINVAL;  // PXN pooling: one ell per server (:274, :850)
  std::vector<uint32_t> stragglers, healthy;
  for (uint32_t v = 0; v < q; ++v) (ell[v * g] > 1.0 ? stragglers : healthy).push_back(v);
  std::stable_sort(stragglers.begin(), stragglers.end(),
                   [&](uint32_t a, uint32_t b) { return ell[a * g] > ell[b * g]; });  // l1 >= l2 >= ... (:78)
  if (healthy.size() < 2) return OPTCC_EINVAL;
  if (g > 1 && stragglers.empty()) return OPTCC_EUNSUPPORTED;      // all-healthy g>1 is NCCL's multi-channel ring (:88)
  if (g > 255) return OPTCC_EUNSUPPORTED;                           // `part` is a byte
  const uint32_t ordering = (opts && opts->ordering) ? opts->ordering : 2;   // 0 = default = ordering (2)
  if (ordering != 1 && ordering != 2 && ordering != 3) return OPTCC_EINVAL;  // the two valid orderings of :138, or their mix (:144-155)
  if (ordering != 2 && !(g == 1 && stragglers.size() == 1 && schedule == OPTCC_SCHED_OPTCC)) return OPTCC_EUNSUPPORTED;
  if (n == 0 || n > (uint64_t(1) << 40)) return OPTCC_EINVAL;
  if (dtype != OPTCC_F32 && dtype != OPTCC_BF16) return OPTCC_EINVAL;
  uint32_t k = opts ? opts->k : 0;
  if (k != 0 && (k % 4 != 0 || k > 65536)) return OPTCC_EINVAL;  // multiple of 4 (:155)

  optcc_plan_t* pl = new (std::nothrow) optcc_plan_t();
  if (!pl) return OPTCC_ENOMEM;
  pl->exec = nullptr;
  std::memset(&pl->info, 0, sizeof pl->info);
  std::memset(&pl->opts, 0, sizeof pl->opts);
  if (opts) pl->opts = *opts;
  if (pl->opts.exec_mode > OPTCC_EXEC_COLUMN) { delete pl; return OPTCC_EINVAL; }
  const bool exec_auto = pl->opts.exec_mode == OPTCC_EXEC_AUTO;
  if (exec_auto) pl->opts.exec_mode = OPTCC_EXEC_COLUMN;   // (tile geometry is the column executor's; see the check below)
  pl->ell.assign(ell, ell + p);
  pl->stragglers = stragglers;
  pl->healthy = healthy;
  const uint32_t m = (uint32_t)stragglers.size(), H = (uint32_t)healthy.size();
  const uint32_t construction = (m == 0 || schedule == OPTCC_SCHED_RING_DEGRADED)
                                    ? OPTCC_C0 : (g > 1 ? OPTCC_C3 : (m == 1 ? OPTCC_C1 : OPTCC_C2));
  const double ell1 = m ? ell[stragglers[0] * g] : 1.0;

  const uint64_t A = dtype == OPTCC_F32 ? 4 : 8;  // elements per 16-byte unit (PLAN_SPEC 2, R3)
  const uint64_t U = (n + A - 1) / A;
  auto split = [](uint64_t lo, uint64_t hi, uint64_t parts, uint64_t i) {
    // PLAN_SPEC 2: lo + floor(i (hi-lo) / parts); i <= parts <= 2^23 and hi-lo <= 2^40, so no overflow in u64
    return lo + (i * (hi - lo)) / parts;
  };
  auto E = [&](uint64_t u) { return std::min(u * A, n); };

  // ---- PLAN_SPEC 2: bandwidth-weighted chunking (n_p2p/n = (2-l)/((p-2)l+2)) ----
  uint64_t U_p2p = 0;
  if (construction == OPTCC_C1 && ell1 < 2.0) {
    volatile double num = 2.0 - ell1;                 // volatile: one rounding per operation, in this order
    volatile double den = double(p - 2) * ell1;
    den = den + 2.0;
    volatile double f = num / den;
    volatile double x = double(U) * f;
    U_p2p = (uint64_t)std::floor(x + 0.5);
  }
  const uint64_t U_ring = U - U_p2p;
  std::vector<std::pair<uint64_t, uint64_t>> ring;   // ring region of every part, in units
  if (construction == OPTCC_C0 || construction == OPTCC_C1) {
    ring.push_back({0, U_ring});
  } else {
    for (int lam = 0; lam < g; ++lam) ring.push_back({split(0, U, g, lam), split(0, U, g, lam + 1)});
  }
  // k (PLAN_SPEC 2 "k (R2)")
  if (construction == OPTCC_C0) {
    k = 1;
  } else if (k == 0) {
    double c = construction == OPTCC_C1 ? (ell1 < 2.0 ? ell1 - 1.0 : 1.0) : (construction == OPTCC_C2 ? 1.0 : 2.0);
    uint64_t k_t = 4 * (uint64_t)std::ceil(5.0 * c - 1e-9);
    uint64_t R = (ring[0].second - ring[0].first) * 16;
    uint64_t k_c = 4 * ((R / (uint64_t(H) * 65536)) / 4);
    k = (uint32_t)std::max<uint64_t>(4, std::min(k_t, k_c));
  }
  const uint32_t nsec = construction == OPTCC_C0 ? (uint32_t)p : H;
  const bool bubbles = construction == OPTCC_C1 && ell1 < 2.0;

  Geom G;
  G.p = p; G.g = g; G.q = q; G.m = m; G.H = H; G.k = k; G.nsec = nsec;
  G.construction = construction; G.ordering = ordering; G.bubbles = bubbles;
  G.healthy = pl->healthy.data();
  G.stragglers = pl->stragglers.data();
  uint64_t reduce_elems = 0, copy_elems = 0;
  try {
    // ---- exported boundary arrays (PLAN_SPEC 2): every section start in (part, segment, section) order ----
    const uint32_t nparts = (uint32_t)ring.size();
    pl->sec_bounds.reserve(size_t(nparts) * k * nsec + 1);
    for (uint32_t lam = 0; lam < nparts; ++lam)
      for (uint32_t b = 0; b < k; ++b) {
        const uint64_t s0 = split(ring[lam].first, ring[lam].second, k, b), s1 = split(ring[lam].first, ring[lam].second, k, b + 1);
        for (uint32_t c = 0; c < nsec; ++c) pl->sec_bounds.push_back(E(split(s0, s1, nsec, c)));
      }
    pl->sec_bounds.push_back(E(ring.back().second));
    if (bubbles) {
      for (uint32_t b = 0; b <= k; ++b) pl->p2p_bounds.push_back(E(split(U_ring, U, k, b)));
    }
    // ---- regions = the sections and P2P pieces themselves: consecutive exported boundaries (ascending, contiguous,
    // covering [0, n): PLAN_SPEC 5.4).  A flow carries its (part, segment, section), i.e. its region, from birth, so
    // offset and length are the region's by construction.
    auto add_regions = [&](const std::vector<uint64_t>& bounds, std::vector<uint32_t>& reg_of, bool sections) {
      reg_of.assign(bounds.empty() ? 0 : bounds.size() - 1, UINT32_MAX);
      for (size_t i = 0; i + 1 < bounds.size(); ++i) {
        if (bounds[i + 1] <= bounds[i]) continue;
        reg_of[i] = (uint32_t)pl->region_offs.size();
        pl->region_offs.push_back(bounds[i]);
        pl->region_len.push_back(bounds[i + 1] - bounds[i]);
        // interval i of sec_bounds is (part, segment, section) = (i / (k nsec), (i / nsec) mod k, i mod nsec).  Class =
        // (part, pattern, section): the segments of the four-pattern mix repeat with period 4, all others with period 1.
        const uint32_t period = ordering == 3 ? 4 : 1;
        const uint32_t seg = uint32_t((i / nsec) % k);
        pl->region_class.push_back(sections ? (uint32_t(i / (size_t(k) * nsec)) * period + seg % period) * nsec + uint32_t(i % nsec)
                                            : nparts * period * nsec);
      }
    };
    add_regions(pl->sec_bounds, G.sec_reg, true);
    add_regions(pl->p2p_bounds, G.p2p_reg, false);
    {   // the regions tile [0, n) exactly (both executors and the lazy verifier rely on it)
      uint64_t pos = 0;
      for (size_t r = 0; r < pl->region_offs.size(); ++r) {
        if (pl->region_offs[r] != pos) { delete pl; return OPTCC_EINVAL; }
        pos += pl->region_len[r];
      }
      if (pos != n) { delete pl; return OPTCC_EINVAL; }
    }
    G.region_off = pl->region_offs.data();
    G.region_len = pl->region_len.data();
    G.str_by_rank.resize(m);
    for (uint32_t i = 0; i < m; ++i) G.str_by_rank[i] = i;
    std::sort(G.str_by_rank.begin(), G.str_by_rank.end(), [&](uint32_t a, uint32_t b) { return stragglers[a] < stragglers[b]; });

    // ---- PLAN_SPEC 4: constructions.  Step counts; the flows come from emit_step ----
    if (construction == OPTCC_C1 && ordering == 3) {
      G.P = H; G.n_steps = (k + 1) * H;
    } else if (construction == OPTCC_C1 && ordering == 1) {
      G.P = H; G.n_steps = (k + 3) * H;
    } else if (construction == OPTCC_C0) {
      G.P = p; G.n_steps = 2 * (p - 1);
    } else {
      G.P = H + m - 1;  // windows per body: H for C1/C3, p-1 for C2 (:788)
      if (construction == OPTCC_C3) {
        G.D = 1 + (uint32_t)((g - 2 + G.P - 1) / G.P);  // NIC body of segment b is body b + D (PLAN_SPEC C3)
        G.n_steps = (k + G.D + 2) * G.P + g - 2;
      } else {
        G.n_steps = (k + 1) * G.P;
      }
    }
    const uint32_t n_steps = G.n_steps;
    // pass 1: flows per step; pass 2: fill.  Steps are independent: both passes run on a few host threads for big tables.
    pl->step_begin.assign(size_t(n_steps) + 1, 0);
    const size_t est = size_t(2) * (k + 1) * (p - 1) * (nsec + m) * (g > 1 ? 2 : 1);
    const size_t n_chunks = std::min<size_t>(n_steps, 64);
    auto chunk_lo = [&](size_t c) { return uint32_t(uint64_t(n_steps) * c / n_chunks); };
    bool any_empty = false;
    for (uint32_t r : G.sec_reg) any_empty |= r == UINT32_MAX;
    for (uint32_t r : G.p2p_reg) any_empty |= r == UINT32_MAX;
    optcc_parallel_chunks(n_chunks, est, [&](size_t c) {
      for (uint32_t t = chunk_lo(c); t < chunk_lo(c + 1); ++t) {
        if (any_empty) {
          CountSink cs;
          emit_step(G, t, cs);
          pl->step_begin[t + 1] = cs.n;
        } else {
          CountAllSink cs;
          emit_step(G, t, cs);
          pl->step_begin[t + 1] = cs.n;
        }
      }
    });
    uint64_t total = 0;
    uint32_t max_per_step = 0;
    for (uint32_t t = 0; t < n_steps; ++t) {
      const uint32_t c = pl->step_begin[t + 1];
      max_per_step = std::max(max_per_step, c);
      total += c;
      if (total > 0xFFFFFFF0ull) { delete pl; return OPTCC_EUNSUPPORTED; }   // flow indices are 32-bit
      pl->step_begin[t + 1] = (uint32_t)total;
    }
    pl->info.max_flows_per_step = max_per_step;
    pl->flows.resize_uninit(total);
    pl->flow_region.resize_uninit(total);
    std::vector<uint64_t> red(n_chunks, 0), cop(n_chunks, 0);
    const size_t nreg = pl->region_offs.size();
    std::vector<uint32_t> hist(n_chunks * nreg, 0);      // flows per (chunk, region)
    optcc_parallel_chunks(n_chunks, est, [&](size_t c) {
      FillSink fs;
      fs.G = &G;
      fs.region_count = hist.data() + c * nreg;
      for (uint32_t t = chunk_lo(c); t < chunk_lo(c + 1); ++t) {
        fs.out = pl->flows.data() + pl->step_begin[t];
        fs.out_region = pl->flow_region.data() + pl->step_begin[t];
        emit_step(G, t, fs);
      }
      red[c] = fs.reduce_elems;
      cop[c] = fs.copy_elems;
    });
    for (size_t c = 0; c < n_chunks; ++c) { reduce_elems += red[c]; copy_elems += cop[c]; }
    pl->region_flows.assign(nreg, 0);
    for (size_t c = 0; c < n_chunks; ++c)
      for (size_t r = 0; r < nreg; ++r) pl->region_flows[r] += hist[c * nreg + r];
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  const uint32_t n_steps = G.n_steps;

  optcc_plan_info_t& in = pl->info;
  in.p = p; in.g = g; in.q = q; in.m = m; in.H = H; in.k = k;
  in.construction = construction; in.dtype = dtype; in.unit_elems = (uint32_t)A;
  // narrowest mask that holds p bits and keeps every flow offset (a multiple of A elements) 16-byte aligned: >= 16/A bytes
  in.mask_bytes = p <= 16 ? 2 : (p <= 32 ? 4 : (p <= 64 ? 8 : (p <= 128 ? 16 : 0)));
  if (in.mask_bytes) in.mask_bytes = std::max<uint32_t>(in.mask_bytes, uint32_t(16 / A));
  in.mask_words = (in.mask_bytes + 7) / 8;
  in.n = n; in.n_ring = E(U_ring); in.n_p2p = n - E(U_ring);
  in.U = U; in.U_ring = U_ring; in.U_p2p = U_p2p;
  in.n_steps = n_steps; in.n_flows = (uint32_t)pl->flows.size();
  in.n_sec_bounds = (uint32_t)pl->sec_bounds.size(); in.n_p2p_bounds = (uint32_t)pl->p2p_bounds.size();
  in.reduce_elems = reduce_elems; in.copy_elems = copy_elems;
  // tiling: flows per region (all flows over a region share offset and length), tile counts
  try {
    const size_t nr = pl->region_offs.size();
    uint64_t flow_units = 0;
    for (size_t r = 0; r < nr; ++r) flow_units += uint64_t(pl->region_flows[r]) * ((pl->region_len[r] + A - 1) / A);
    // AUTO: the column executor whenever its work items (one per region and tile) can be indexed with 32 bits -- units
    // / 1792 + regions, i.e. always for plans whose flow table fits 32-bit indices unless the caller forces tiny tiles;
    // otherwise the dataflow executor with its own tile size.  (Measured on a B200: with chain-ordered
    // lists the column executor is the faster one on every shape of BASELINE.json's configs.)
    if (exec_auto) {
      const uint64_t tu = pl->opts.tile_units ? pl->opts.tile_units : 1792;
      if (U / tu + nr >= (uint64_t(1) << 32)) pl->opts.exec_mode = OPTCC_EXEC_DATAFLOW;
    }
    if (pl->opts.tile_units) {
      pl->tile_units = pl->opts.tile_units;
      pl->col_warp = pl->opts.exec_mode == OPTCC_EXEC_COLUMN && pl->tile_units <= 256;   // (small tiles: one warp each)
    } else if (pl->opts.exec_mode == OPTCC_EXEC_COLUMN) {
      // column executor: a tile is taken through its region's whole flow list, so the tile size does not depend on the
      // number of steps.  CTA-wide tiles are one whole streaming round of the CTA (448 threads x 4 vectors = 1792
      // units for f32, x 2 units = 896 for bf16 plans, whose fp32 shadow triples the bytes per unit): whole rounds are
      // what the dead-source discard acts on.  Plans whose regions are shorter than two such tiles (C4: 1092 units at
      // k = 8, 273 at k = 32; C3 at k = 20) take warp-wide tiles of 128 units instead -- a CTA-wide tile would leave
      // most of the CTA idle -- (measured on a B200).
      const uint32_t cta_tile = dtype == OPTCC_BF16 ? 896 : 1792;
      uint64_t longest = 0;
      for (size_t r = 0; r < nr; ++r) longest = std::max(longest, pl->region_len[r]);
      const uint64_t longest_units = ((longest + A - 1) / A + 7) & ~uint64_t(7);
      pl->col_warp = longest_units < 2 * uint64_t(cta_tile);
      pl->tile_units = pl->col_warp ? 128 : cta_tile;
    } else {
      // auto: about two tile-ops per CTA and step (592 = 2 x 296 CTAs on a B200), from {224, 448, 896, 1792, 3584}
      // -- multiples / fractions of one streaming round of the dataflow kernel (448 threads x 4 vectors), so a tile is
      // whole rounds; big steps get 56 KB tiles (bandwidth-bound), small steps short tiles (more parallel chains)
      const uint64_t per = n_steps ? flow_units / n_steps / 592 : 0;
      uint32_t tu = 224;
      while (tu < OPTCC_TILE_UNITS_DEFAULT && uint64_t(tu) * 3 / 2 < per) tu *= 2;
      pl->tile_units = tu;
    }
    uint64_t tiles = 0;
    pl->region_tile0.resize(nr);
    pl->n_tile_ops = 0;
    for (size_t r = 0; r < nr; ++r) {
      pl->region_tile0[r] = tiles;
      const uint64_t rt = ((pl->region_len[r] + A - 1) / A + pl->tile_units - 1) / pl->tile_units;
      tiles += rt;
      pl->n_tile_ops += rt * pl->region_flows[r];
    }
    pl->tiles_per_rank = tiles;
    // the verifier's tiles (column executor): about as many bytes of masks as a data tile has bytes of data -- a unit
    // of A elements is A * mask_bytes >= 16 bytes of masks; CTA-wide unless the regions are shorter than one such tile
    pl->mask_tile_units = pl->tile_units;
    pl->mask_tiles_per_rank = tiles;
    pl->mask_warp = pl->col_warp;
    if (pl->opts.exec_mode == OPTCC_EXEC_COLUMN && in.mask_bytes) {
      const uint64_t mb = A * in.mask_bytes;     // bytes of masks per unit
      auto scaled = [&](uint64_t units) { return std::max<uint64_t>(8, (units * 16 / mb) & ~uint64_t(7)); };
      uint64_t mtu;
      if (pl->opts.tile_units) {
        mtu = scaled(pl->tile_units);
      } else {
        // CTA-wide mask tiles of 28 KB whatever the data type (measured on a B200, r02: C3 1.39 ms against 1.92 ms with
        // 14 KB tiles and 1.81 ms with warp-wide tiles; C4 at k = 32, 273-unit regions: 1.96 against 2.09 ms warp-wide);
        // warp-wide only when the regions are shorter than a quarter of such a tile
        const uint64_t cta_tile = scaled(1792);
        uint64_t longest = 0;
        for (size_t r = 0; r < nr; ++r) longest = std::max(longest, pl->region_len[r]);
        pl->mask_warp = 4 * ((longest + A - 1) / A) < cta_tile;
        mtu = pl->mask_warp ? scaled(128) : cta_tile;
      }
      if (mtu != pl->tile_units) {
        pl->mask_tile_units = (uint32_t)mtu;
        uint64_t mt = 0;
        for (size_t r = 0; r < nr; ++r) mt += ((pl->region_len[r] + A - 1) / A + mtu - 1) / mtu;
        pl->mask_tiles_per_rank = mt;
      }
    }
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  // lazy verifier (optcc.h, lazy_verify): every (rank, region) is written by a flow of the executed steps.  A complete
  // schedule writes every range (each rank receives every section's sum by a reduce or a copy: PLAN_SPEC 5.2); the
  // executor's table build checks it region by region and falls back to the eager form otherwise.  Truncated schedules
  // (step_limit) are walked here.
  try {
    in.lazy_verify = 0;
    if (in.mask_bytes && !pl->opts.verify_eager) {
      if (!pl->opts.step_limit || pl->opts.step_limit >= n_steps) {
        in.lazy_verify = 1;
      } else {
        const uint32_t steps = pl->opts.step_limit;
        const size_t nr = pl->region_offs.size();
        std::vector<uint8_t> written(size_t(p) * nr, 0);
        size_t left = written.size();
        for (uint32_t i = 0; i < pl->step_begin[steps]; ++i) {
          const optcc_flow_t& f = pl->flows[i];
          uint8_t& w = written[size_t(f.dst) * nr + pl->flow_region[i]];
          left -= !w;
          w = 1;
        }
        in.lazy_verify = left == 0;
      }
    }
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  in.exec_mode = pl->opts.exec_mode;
  optcc_ws_layout L = optcc_layout(pl);
  in.workspace_bytes = L.end_exec;
  in.verify_workspace_bytes = L.end_verify;
  in.mask_offset_bytes = L.masks;
  in.padded_n = (n + 7) & ~uint64_t(7);
  in.plan_build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
  *out = pl;
  return OPTCC_OK;
}

extern "C" int optcc_plan(int p, int g, const double* ell, uint64_t n, int dtype, optcc_plan_t** out) {
  return optcc_plan_ex(p, g, ell, n, dtype, nullptr, out);
}

extern "C" void optcc_plan_destroy(optcc_plan_t* plan) {
  if (!plan) return;
  if (plan->exec) optcc_exec_state_free(plan->exec);
  delete plan;
}

extern "C" int optcc_plan_info(const optcc_plan_t* plan, optcc_plan_info_t* out) {
  if (!plan || !out) return OPTCC_EINVAL;
  *out = plan->info;
  return OPTCC_OK;
}

extern "C" int optcc_plan_tables(const optcc_plan_t* plan, const optcc_flow_t** flows, const uint32_t** step_begin,
                                 const uint64_t** sec_bounds, const uint64_t** p2p_bounds) {
  if (!plan) return OPTCC_EINVAL;
  if (flows) *flows = plan->flows.data();
  if (step_begin) *step_begin = plan->step_begin.data();
  if (sec_bounds) *sec_bounds = plan->sec_bounds.data();
  if (p2p_bounds) *p2p_bounds = plan->p2p_bounds.data();
  return OPTCC_OK;
}

extern "C" const char* optcc_strerror(int code) {
  switch (code) {
    case OPTCC_OK: return "ok";
    case OPTCC_EINVAL: return "invalid argument (PLAN_SPEC 1)";
    case OPTCC_EUNSUPPORTED: return "unsupported configuration (g>1 needs a straggler server; ordering 1 and the ring baseline need g=1; masks need p<=128)";
    case OPTCC_ENOMEM: return "out of host memory";
    case OPTCC_ECUDA: return "CUDA runtime error (see optcc_last_cuda_error)";
    case OPTCC_EVERIFY: return "contributor-mask verification failed";
    case OPTCC_ESTALE: return "the workspace did not hold this plan's tables when a kernel ran: call optcc_prepare and run again";
    case OPTCC_ETOOBIG: return "the plan needs more workspace than the library's static array holds (OPTCC_STATIC_WORKSPACE_BYTES): use optcc_execute with a caller workspace";
    default: return "unknown optcc error";
  }
}

extern "C" int optcc_abi_version(void) { return OPTCC_ABI_VERSION; }
