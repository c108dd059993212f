// Host planner of liboptcc: builds the ell-weighted stage / chunk / step plan of OPTCC.
//
// Written from docs/PLAN_SPEC.md (which freezes the canonical reading of PAPER.md 4.1-4.4, App. C/D/E) and the
// paper itself; citations are PAPER.md:<line>.  Pure host C++, no CUDA: closed-form rules, O(p k) flows
// ("closed-form rules ... O(pk)").  Compiled with -ffp-contract=off: the one floating-point
// quantity that decides integers (the P2P share, PLAN_SPEC 2) must round exactly as the spec says.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <atomic>
#include <thread>
#include <new>

#include "optcc_internal.h"

namespace {

struct Builder {
  optcc_plan_t* pl;
  uint64_t A, U, n;
  uint32_t k, nsec;
  std::vector<std::pair<uint64_t, uint64_t>> ring;  // ring region of every part, in units

  static uint64_t split(uint64_t lo, uint64_t hi, uint64_t parts, uint64_t i) {
    // PLAN_SPEC 2: lo + floor(i (hi-lo) / parts); i <= parts <= 2^23 and hi-lo <= 2^40, so no overflow in u64
    return lo + (i * (hi - lo)) / parts;
  }
  uint64_t E(uint64_t u) const { return std::min(u * A, n); }
  std::vector<uint64_t> sec_tab;   // section boundaries [(lam * k + b) * (nsec + 1) + c], filled once by build_sec_tab
  void build_sec_tab() {
    sec_tab.resize(ring.size() * size_t(k) * (nsec + 1));
    for (size_t lam = 0; lam < ring.size(); ++lam)
      for (uint32_t b = 0; b < k; ++b) {
        const uint64_t s0 = split(ring[lam].first, ring[lam].second, k, b);
        const uint64_t s1 = split(ring[lam].first, ring[lam].second, k, b + 1);
        uint64_t* row = sec_tab.data() + (lam * k + b) * (nsec + 1);
        for (uint32_t c = 0; c <= nsec; ++c) row[c] = split(s0, s1, nsec, c);
      }
  }
  void sec_units(uint32_t lam, uint32_t b, uint32_t c, uint64_t* lo, uint64_t* hi) const {
    const uint64_t* row = sec_tab.data() + (size_t(lam) * k + b) * (nsec + 1);
    *lo = row[c];
    *hi = row[c + 1];
  }
  void emit_units(uint32_t step, uint8_t op, uint8_t stage, uint8_t link, uint32_t part, uint32_t src,
                  uint32_t dst, uint32_t seg, uint32_t sec, uint64_t ulo, uint64_t uhi) {
    uint64_t off = E(ulo), len = E(uhi) - E(ulo);
    if (len == 0) return;  // PLAN_SPEC 2: zero-length flows are dropped
    optcc_flow_t f;
    std::memset(&f, 0, sizeof f);
    f.off = off; f.len = len; f.step = step; f.seg = seg; f.sec = sec;
    f.src = (uint16_t)src; f.dst = (uint16_t)dst; f.op = op; f.stage = stage; f.link = link; f.part = (uint8_t)part;
    pl->flows.push_back(f);
  }
  void emit_sec(uint32_t step, uint8_t op, uint8_t stage, uint8_t link, uint32_t lam, uint32_t src, uint32_t dst,
                uint32_t b, uint32_t c) {
    uint64_t lo, hi;
    sec_units(lam, b, c, &lo, &hi);
    emit_units(step, op, stage, link, lam, src, dst, b, c, lo, hi);
  }
};

inline uint32_t modH(int64_t x, int64_t H) { int64_t r = x % H; return (uint32_t)(r < 0 ? r + H : r); }

// Run body(i) for i in [0, n) on a few host threads when the table is large enough to pay for them; the
// iterations are independent (each sorts or moves a disjoint range).
template <class F>
void parallel_chunks(size_t n, size_t work, F body) {
  unsigned hw = std::thread::hardware_concurrency();
  unsigned nt = work < (size_t(1) << 17) ? 1u : std::min(8u, hw ? hw : 1u);
  if (nt <= 1 || n <= 1) { for (size_t i = 0; i < n; ++i) body(i); return; }
  std::atomic<size_t> next{0};
  auto worker = [&]() { for (size_t i; (i = next.fetch_add(1, std::memory_order_relaxed)) < n;) body(i); };
  std::vector<std::thread> th;
  th.reserve(nt - 1);
  for (unsigned t = 1; t < nt; ++t) th.emplace_back(worker);
  worker();
  for (auto& t : th) t.join();
}

// PLAN_SPEC 3 order (step, link, stage, src, dst, off): counting sort by step, then each step's few flows by a
// packed key -- the table has O(p k H) records, a comparison sort of whole records dominated the build time.
// The per-step sorts and the final gather touch disjoint ranges and are split over host threads.
void sort_flows(std::vector<optcc_flow_t>& flows, uint32_t n_steps) {
  struct Key { uint64_t hi, lo; uint32_t idx; };
  const size_t nf = flows.size();
  std::vector<uint32_t> begin(size_t(n_steps) + 2, 0);
  for (const auto& f : flows) begin[f.step + 1]++;
  for (size_t t = 0; t <= n_steps; ++t) begin[t + 1] += begin[t];
  std::vector<Key> keys(nf);
  {
    std::vector<uint32_t> pos(begin.begin(), begin.end() - 1);
    for (size_t i = 0; i < nf; ++i) {
      const optcc_flow_t& f = flows[i];
      Key k;
      k.hi = (uint64_t(f.link) << 35) | (uint64_t(f.stage) << 32) | (uint64_t(f.src) << 16) | uint64_t(f.dst);
      k.lo = f.off;
      k.idx = (uint32_t)i;
      keys[pos[f.step]++] = k;
    }
  }
  std::vector<optcc_flow_t> out(nf);
  parallel_chunks(size_t(n_steps) + 1, nf, [&](size_t t) {
    std::sort(keys.begin() + begin[t], keys.begin() + begin[t + 1],
              [](const Key& a, const Key& b) { return a.hi != b.hi ? a.hi < b.hi : a.lo < b.lo; });
    for (size_t i = begin[t]; i < begin[t + 1]; ++i) out[i] = flows[keys[i].idx];
  });
  flows.swap(out);
}

// Storage kinds for bf16 plans: walk the table once with the number of contributors every
// (rank, region) holds.  A region holding 1 or all p contributors lives in the rank buffer (bf16); a partial
// sum (1 < count < p) lives in the fp32 shadow.  All flows of one step read the state before the step.
void assign_kinds(optcc_plan_t* pl) {
  const uint32_t p = pl->info.p;
  const size_t nf = pl->flows.size();
  pl->kind_src.assign(nf, OPTCC_KIND_BUF);
  pl->kind_dst_in.assign(nf, OPTCC_KIND_BUF);
  pl->kind_dst_out.assign(nf, OPTCC_KIND_BUF);
  if (pl->info.dtype != OPTCC_BF16) return;
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

}  // namespace

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
  if (ordering != 1 && ordering != 2) return OPTCC_EINVAL;                   // the two valid orderings of :138
  if (ordering == 1 && !(g == 1 && stragglers.size() == 1 && schedule == OPTCC_SCHED_OPTCC)) return OPTCC_EUNSUPPORTED;
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
  else pl->opts.exec_mode = OPTCC_EXEC_DATAFLOW;   // the default executor
  pl->ell.assign(ell, ell + p);
  pl->stragglers = stragglers;
  pl->healthy = healthy;
  const uint32_t m = (uint32_t)stragglers.size(), H = (uint32_t)healthy.size();
  const uint32_t construction = (m == 0 || schedule == OPTCC_SCHED_RING_DEGRADED)
                                    ? OPTCC_C0 : (g > 1 ? OPTCC_C3 : (m == 1 ? OPTCC_C1 : OPTCC_C2));
  const double ell1 = m ? ell[stragglers[0] * g] : 1.0;

  Builder B;
  B.pl = pl;
  B.n = n;
  B.A = dtype == OPTCC_F32 ? 4 : 8;  // elements per 16-byte unit (PLAN_SPEC 2, R3)
  B.U = (n + B.A - 1) / B.A;
  const uint64_t U = B.U;

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
  if (construction == OPTCC_C0 || construction == OPTCC_C1) {
    B.ring.push_back({0, U_ring});
  } else {
    for (int lam = 0; lam < g; ++lam) B.ring.push_back({Builder::split(0, U, g, lam), Builder::split(0, U, g, lam + 1)});
  }
  // k (PLAN_SPEC 2 "k (R2)")
  if (construction == OPTCC_C0) {
    k = 1;
  } else if (k == 0) {
    double c = construction == OPTCC_C1 ? (ell1 < 2.0 ? ell1 - 1.0 : 1.0) : (construction == OPTCC_C2 ? 1.0 : 2.0);
    uint64_t k_t = 4 * (uint64_t)std::ceil(5.0 * c - 1e-9);
    uint64_t R = (B.ring[0].second - B.ring[0].first) * 16;
    uint64_t k_c = 4 * ((R / (uint64_t(H) * 65536)) / 4);
    k = (uint32_t)std::max<uint64_t>(4, std::min(k_t, k_c));
  }
  B.k = k;
  B.nsec = construction == OPTCC_C0 ? (uint32_t)p : H;
  auto p2p_lo = [&](uint32_t b) { return Builder::split(U_ring, U, k, b); };
  try {
    B.build_sec_tab();
    // flows: 2 (p-1) n elements in sections of about U / (g k nsec) units
    pl->flows.reserve(size_t(2) * (k + 1) * (p - 1) * (B.nsec + m) * (g > 1 ? 2 : 1));
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  const bool bubbles = construction == OPTCC_C1 && ell1 < 2.0;

  // ---- PLAN_SPEC 4: constructions ----
  uint32_t n_steps = 0;
  try {
    if (construction == OPTCC_C1 && ordering == 1) {
      // C1': ordering (1) of :138, S1 -> S2 -> S3 -> S4, one stage per body (PLAN_SPEC 4 C1')
      n_steps = (k + 3) * H;
      const uint32_t sg = stragglers[0];
      for (uint32_t Bd = 0; Bd < k + 3; ++Bd) {
        const uint32_t base = Bd * H;
        for (uint32_t j = 0; j < H; ++j) {
          const uint32_t src = healthy[j], dst = healthy[(j + 1) % H];
          for (uint32_t t = 0; t + 1 < H; ++t) {
            const uint32_t step = base + (t < j ? t : t + 1);
            const uint32_t c = modH(int64_t(j) - t, H);
            if (Bd < k)    // Stage 1: partial sums of the healthy servers (:126)
              B.emit_sec(step, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, 0, src, dst, Bd, c);
            if (Bd >= 3)   // Stage 4: the all-gather of section c starts at healthy c (:136)
              B.emit_sec(step, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, 0, src, dst, Bd - 3, c);
          }
        }
        for (uint32_t a = 0; a < H; ++a) {
          const uint32_t d = (a + 1) % H, step = base + a;
          if (Bd >= 1 && Bd <= k)       // Stage 2: the straggler adds its own data to the uploaded partial sum (:130-132)
            B.emit_sec(step, OPTCC_OP_REDUCE, OPTCC_S2, OPTCC_LINK_NIC, 0, healthy[a], sg, Bd - 1, (a + 1) % H);
          if (Bd >= 2 && Bd <= k + 1)   // Stage 3: the global sum returns to the uploader's ring successor (:132, R11)
            B.emit_sec(step, OPTCC_OP_COPY, OPTCC_S3, OPTCC_LINK_NIC, 0, sg, healthy[d], Bd - 2, d);
          if (bubbles && Bd < k)
            B.emit_units(step, OPTCC_OP_REDUCE, OPTCC_BUB_UP, OPTCC_LINK_NIC, 0, healthy[a], sg, Bd, 0, p2p_lo(Bd), p2p_lo(Bd + 1));
          if (bubbles && Bd >= 1 && Bd <= k)
            B.emit_units(step, OPTCC_OP_COPY, OPTCC_BUB_DOWN, OPTCC_LINK_NIC, 0, sg, healthy[d], Bd - 1, 0, p2p_lo(Bd - 1), p2p_lo(Bd));
        }
      }
    } else if (construction == OPTCC_C0) {
      // plain ring: reduce-scatter p-1 hops then all-gather p-1 hops (:52, :72)
      n_steps = 2 * (p - 1);
      for (int t = 0; t < p - 1; ++t)
        for (int j = 0; j < p; ++j) {
          uint32_t d = (j + 1) % p;
          B.emit_sec(t, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, 0, j, d, 0, modH(j - t, p));
          B.emit_sec(p - 1 + t, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, 0, j, d, 0, modH(j + 1 - t, p));
        }
    } else {
      const uint32_t P = H + m - 1;  // windows per body: H for C1/C3, p-1 for C2 (:788)
      uint32_t D = 0;
      if (construction == OPTCC_C3) {
        D = 1 + (uint32_t)((g - 2 + P - 1) / P);  // NIC body of segment b is body b + D (PLAN_SPEC C3)
        n_steps = (k + D + 2) * P + g - 2;
      } else {
        n_steps = (k + 1) * P;
      }
      for (int lam = 0; lam < g; ++lam) {
        // leaders: local GPU lam of every server (:854); for g = 1 simply the ranks
        for (uint32_t Bd = 0; Bd <= k; ++Bd) {
          const uint32_t base = (Bd + D) * P;
          // ring link j (healthy j -> j+1) is idle in windows [j, j+m); hop t sits in window W(j,t)
          for (uint32_t j = 0; j < H; ++j) {
            uint32_t src = healthy[j] * g + lam, dst = healthy[(j + 1) % H] * g + lam;
            for (uint32_t t = 0; t + 1 < H; ++t) {
              uint32_t step = base + (t < j ? t : t + m);
              if (Bd < k)   // Stage 1, hop t of segment Bd: add own section and forward (:126)
                B.emit_sec(step, OPTCC_OP_REDUCE, OPTCC_S1, OPTCC_LINK_NIC, lam, src, dst, Bd, modH(int64_t(j) - t, H));
              if (Bd >= 1)  // Stage 4, hop t of segment Bd-1: forward the complete sum (:136)
                B.emit_sec(step, OPTCC_OP_COPY, OPTCC_S4, OPTCC_LINK_NIC, lam, src, dst, Bd - 1, modH(int64_t(j) + 1 - t, H));
            }
          }
          for (uint32_t i = 0; i < m; ++i) {
            uint32_t sg = stragglers[i] * g + lam;
            for (uint32_t a = 0; a < H; ++a) {
              uint32_t d = (a + 1) % H, step = base + a + i;
              uint32_t ra = healthy[a] * g + lam, rd = healthy[d] * g + lam;
              if (Bd >= 1)  // Stage 2: the owner uploads the complete sum to the straggler (:130; ordering (2) :138)
                B.emit_sec(step, OPTCC_OP_COPY, OPTCC_S2, OPTCC_LINK_NIC, lam, ra, sg, Bd - 1, (a + 1) % H);
              if (Bd < k)   // Stage 3: the straggler's raw section is folded in at its owner (:132, :138)
                B.emit_sec(step, OPTCC_OP_REDUCE, OPTCC_S3, OPTCC_LINK_NIC, lam, sg, rd, Bd, (d + 1) % H);
              if (bubbles && Bd < k)   // bubble-up: healthy a's raw P2P piece into the straggler (:165, R9)
                B.emit_units(step, OPTCC_OP_REDUCE, OPTCC_BUB_UP, OPTCC_LINK_NIC, lam, ra, sg, Bd, 0, p2p_lo(Bd), p2p_lo(Bd + 1));
              if (bubbles && Bd >= 1)  // bubble-down: the straggler returns the P2P result (:165)
                B.emit_units(step, OPTCC_OP_COPY, OPTCC_BUB_DOWN, OPTCC_LINK_NIC, lam, sg, rd, Bd - 1, 0, p2p_lo(Bd - 1), p2p_lo(Bd));
            }
          }
        }
        if (construction == OPTCC_C3) {
          for (uint32_t v = 0; v < q; ++v)
            for (uint32_t b = 0; b < k; ++b)
              for (uint32_t c = 0; c < H; ++c)
                for (int h = 0; h + 1 < g; ++h) {
                  // N1/N3 collect on the backward local ring, the leader only receives (:862, :875, :894)
                  B.emit_sec(b * P + c + h, OPTCC_OP_REDUCE, OPTCC_N_COLLECT, OPTCC_LINK_NVLINK, lam,
                             v * g + modH(lam - 1 - h, g), v * g + modH(lam - 2 - h, g), b, c);
                  // N2/N4 distribute on the forward local ring, the leader sends first (:863, :876, :894)
                  B.emit_sec((b + D + 2) * P + c + h, OPTCC_OP_COPY, OPTCC_N_DISTRIBUTE, OPTCC_LINK_NVLINK, lam,
                             v * g + modH(lam + h, g), v * g + modH(lam + h + 1, g), b, c);
                }
        }
      }
    }
    sort_flows(pl->flows, n_steps);
    pl->step_begin.assign(n_steps + 1, 0);
    {
      size_t i = 0;
      for (uint32_t t = 0; t <= n_steps; ++t) {
        while (i < pl->flows.size() && pl->flows[i].step < t) ++i;
        pl->step_begin[t] = (uint32_t)i;
      }
    }
    // exported boundary arrays (PLAN_SPEC 2)
    uint32_t nparts = (construction == OPTCC_C2 || construction == OPTCC_C3) ? (uint32_t)g : 1;
    for (uint32_t lam = 0; lam < nparts; ++lam)
      for (uint32_t b = 0; b < k; ++b)
        for (uint32_t c = 0; c < B.nsec; ++c) {
          uint64_t lo, hi;
          B.sec_units(lam, b, c, &lo, &hi);
          pl->sec_bounds.push_back(B.E(lo));
        }
    pl->sec_bounds.push_back(B.E(B.ring.back().second));
    if (bubbles) {
      for (uint32_t b = 0; b < k; ++b) pl->p2p_bounds.push_back(B.E(p2p_lo(b)));
      pl->p2p_bounds.push_back(B.E(U));
    }
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }

  optcc_plan_info_t& in = pl->info;
  in.p = p; in.g = g; in.q = q; in.m = m; in.H = H; in.k = k;
  in.construction = construction; in.dtype = dtype; in.unit_elems = (uint32_t)B.A;
  // narrowest mask that holds p bits and keeps every flow offset (a multiple of A elements) 16-byte aligned: >= 16/A bytes
  in.mask_bytes = p <= 16 ? 2 : (p <= 32 ? 4 : (p <= 64 ? 8 : (p <= 128 ? 16 : 0)));
  if (in.mask_bytes) in.mask_bytes = std::max<uint32_t>(in.mask_bytes, uint32_t(16 / B.A));
  in.mask_words = (in.mask_bytes + 7) / 8;
  in.n = n; in.n_ring = B.E(U_ring); in.n_p2p = n - B.E(U_ring);
  in.U = U; in.U_ring = U_ring; in.U_p2p = U_p2p;
  in.n_steps = n_steps; in.n_flows = (uint32_t)pl->flows.size();
  in.n_sec_bounds = (uint32_t)pl->sec_bounds.size(); in.n_p2p_bounds = (uint32_t)pl->p2p_bounds.size();
  for (uint32_t t = 0; t < n_steps; ++t)
    in.max_flows_per_step = std::max(in.max_flows_per_step, pl->step_begin[t + 1] - pl->step_begin[t]);
  for (const auto& f : pl->flows) (f.op == OPTCC_OP_REDUCE ? in.reduce_elems : in.copy_elems) += f.len;
  // dataflow tiling: regions (unique offsets; all flows over one offset share a length, PLAN_SPEC 5.4) and tile counts
  try {
    if (pl->opts.tile_units) {
      pl->tile_units = pl->opts.tile_units;
    } else if (pl->opts.exec_mode == OPTCC_EXEC_COLUMN) {
      // column executor: a CTA runs a region's whole flow list on one tile, so the tile size does not depend on the
      // number of steps.  One whole streaming round of the CTA (448 threads x 4 vectors = 1792 units for f32, x 2
      // units = 896 for bf16 plans, whose fp32 shadow triples the bytes per unit): whole rounds are what the
      // dead-source discard acts on (measured on a B200); a region shorter than that is one tile.
      uint32_t tu = dtype == OPTCC_BF16 ? 896 : 1792;
      uint64_t longest = 0;
      for (size_t i = 0; i + 1 < pl->sec_bounds.size(); ++i) longest = std::max(longest, pl->sec_bounds[i + 1] - pl->sec_bounds[i]);
      for (size_t i = 0; i + 1 < pl->p2p_bounds.size(); ++i) longest = std::max(longest, pl->p2p_bounds[i + 1] - pl->p2p_bounds[i]);
      const uint64_t longest_units = ((longest + B.A - 1) / B.A + 7) & ~uint64_t(7);
      if (longest_units && longest_units < tu) tu = (uint32_t)longest_units;
      pl->tile_units = tu;
    } else {
      // auto: about two tile-ops per CTA and step (592 = 2 x 296 CTAs on a B200), from {224, 448, 896, 1792, 3584}
      // -- multiples / fractions of one streaming round of the dataflow kernel (448 threads x 4 vectors), so a tile is
      // whole rounds; big steps get 56 KB tiles (bandwidth-bound), small steps short tiles (more parallel chains)
      uint64_t units = 0;
      for (const auto& f : pl->flows) units += (f.len + B.A - 1) / B.A;
      const uint64_t per = n_steps ? units / n_steps / 592 : 0;
      uint32_t tu = 224;
      while (tu < OPTCC_TILE_UNITS_DEFAULT && uint64_t(tu) * 3 / 2 < per) tu *= 2;
      pl->tile_units = tu;
    }
    // regions = the sections and P2P pieces themselves: consecutive exported boundaries (ascending, contiguous)
    uint64_t tiles = 0;
    std::vector<uint32_t> sec_reg, p2p_reg;     // boundary interval -> region (UINT32_MAX: empty interval)
    bool region_error = false;
    auto add_regions = [&](const std::vector<uint64_t>& bounds, std::vector<uint32_t>& reg_of) {
      reg_of.assign(bounds.empty() ? 0 : bounds.size() - 1, UINT32_MAX);
      for (size_t i = 0; i + 1 < bounds.size(); ++i) {
        if (bounds[i + 1] <= bounds[i]) continue;
        reg_of[i] = (uint32_t)pl->region_offs.size();
        pl->region_offs.push_back(bounds[i]);
        pl->region_tile0.push_back(tiles);
        tiles += ((bounds[i + 1] - bounds[i] + B.A - 1) / B.A + pl->tile_units - 1) / pl->tile_units;
      }
    };
    add_regions(pl->sec_bounds, sec_reg);
    add_regions(pl->p2p_bounds, p2p_reg);
    pl->tiles_per_rank = tiles;
    // region of every flow, looked up once (the executor's and the cost model's table walks all need it): a flow
    // carries its (part, segment, section), i.e. its interval of sec_bounds (bubble flows: of p2p_bounds)
    pl->flow_region.resize(pl->flows.size());
    {
      const std::vector<uint64_t>& ro = pl->region_offs;
      for (size_t i = 0; i < pl->flows.size(); ++i) {
        const optcc_flow_t& f = pl->flows[i];
        uint32_t r = UINT32_MAX;
        if (f.stage == OPTCC_BUB_UP || f.stage == OPTCC_BUB_DOWN) {
          if (f.seg < p2p_reg.size()) r = p2p_reg[f.seg];
        } else {
          const size_t idx = (size_t(f.part) * k + f.seg) * B.nsec + f.sec;
          if (idx < sec_reg.size()) r = sec_reg[idx];
        }
        if (r == UINT32_MAX || ro[r] != f.off) r = uint32_t(std::lower_bound(ro.begin(), ro.end(), f.off) - ro.begin());
        if (r >= ro.size() || ro[r] != f.off) { region_error = true; break; }   // PLAN_SPEC 5.4 violated: a planner bug
        pl->flow_region[i] = r;
      }
    }
    if (region_error) {
      delete pl;
      return OPTCC_EINVAL;
    }
    for (const auto& f : pl->flows) pl->n_tile_ops += ((f.len + B.A - 1) / B.A + pl->tile_units - 1) / pl->tile_units;
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  try {
    assign_kinds(pl);      // (needs flow_region)
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
  // lazy verifier (optcc.h, lazy_verify): every (rank, region) is written by a flow of the executed steps
  try {
    in.lazy_verify = 0;
    if (in.mask_bytes && !pl->opts.verify_eager) {
      const uint32_t steps = pl->opts.step_limit ? std::min(pl->opts.step_limit, n_steps) : n_steps;
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
  } catch (const std::bad_alloc&) {
    delete pl;
    return OPTCC_ENOMEM;
  }
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
    default: return "unknown optcc error";
  }
}

extern "C" int optcc_abi_version(void) { return OPTCC_ABI_VERSION; }
