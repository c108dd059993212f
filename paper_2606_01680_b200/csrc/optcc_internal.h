// Internal definitions shared by the host planner (optcc_plan.cpp) and the executor (optcc_exec.cu).
// Not part of the ABI.  Nothing here is shared with oracle/ (the oracle is Python and never includes this).
#ifndef OPTCC_INTERNAL_H_
#define OPTCC_INTERNAL_H_

#include <algorithm>
#include <cstddef>
#include <cstdint>
#include <new>
#include <vector>

#include "optcc.h"

// Storage kind of a (rank, region) at some point of a bf16 plan (partial sums stay fp32 between
// steps, one RNE rounding when the sum over all p ranks completes).
enum : uint8_t { OPTCC_KIND_BUF = 0 /* the rank buffer, plan dtype */, OPTCC_KIND_F32 = 1 /* fp32 shadow */ };

struct optcc_exec_state;  // device-side cache, defined in optcc_exec.cu

// Big host tables (the flow table and what is derived from it: tens to hundreds of MB at p = 128 ... 1024).  Memory
// comes uninitialised (every element is written by the fill pass, so no zeroing pass and no single-threaded page faults)
// and goes back to a small process-wide cache when the plan dies: a job that plans every step (bench.py does) gets
// pages that are already mapped.  optcc_raw_alloc / optcc_raw_free live in optcc_plan.cpp.
void* optcc_raw_alloc(size_t bytes);          // nullptr on failure; 64-byte aligned
void optcc_raw_free(void* p, size_t bytes);
template <class T>
class optcc_rawvec {
 public:
  optcc_rawvec() = default;
  optcc_rawvec(const optcc_rawvec&) = delete;
  optcc_rawvec& operator=(const optcc_rawvec&) = delete;
  ~optcc_rawvec() { release(); }
  void release() { if (p_) optcc_raw_free(p_, cap_ * sizeof(T)); p_ = nullptr; n_ = cap_ = 0; }
  void resize_uninit(size_t n) {          // contents undefined; throws std::bad_alloc
    if (n > cap_) {
      release();
      p_ = static_cast<T*>(optcc_raw_alloc(n * sizeof(T)));
      if (!p_) throw std::bad_alloc();
      cap_ = n;
    }
    n_ = n;
  }
  size_t size() const { return n_; }
  bool empty() const { return n_ == 0; }
  T* data() { return p_; }
  const T* data() const { return p_; }
  T& operator[](size_t i) { return p_[i]; }
  const T& operator[](size_t i) const { return p_[i]; }
  T* begin() { return p_; }
  T* end() { return p_ + n_; }
  const T* begin() const { return p_; }
  const T* end() const { return p_ + n_; }
 private:
  T* p_ = nullptr;
  size_t n_ = 0, cap_ = 0;
};

struct optcc_plan {
  optcc_plan_info_t info;
  optcc_opts_t opts;
  std::vector<double> ell;              // [p]
  std::vector<uint32_t> stragglers;     // server indices, ell descending then index (PLAN_SPEC 1)
  std::vector<uint32_t> healthy;        // server indices ascending
  optcc_rawvec<optcc_flow_t> flows;     // in PLAN_SPEC 3 order
  std::vector<uint32_t> step_begin;     // [n_steps + 1]
  std::vector<uint64_t> sec_bounds;
  std::vector<uint64_t> p2p_bounds;
  // per flow, bf16 plans only: storage kinds of src, dst before, dst after (host walk over contributor counts)
  std::vector<uint8_t> kind_src, kind_dst_in, kind_dst_out;
  // dataflow executor (exec_mode 2): every flow is cut into tiles of `tile_units` 16-byte units; tile-ops are
  // claimed in table order and wait on per-(rank, region, tile) completion counters instead of a grid barrier
  uint32_t tile_units = 0;
  uint64_t n_tile_ops = 0;              // sum over flows of ceil(units / tile_units)
  uint64_t tiles_per_rank = 0;          // sum over regions of ceil(units / tile_units): counters per rank
  // column executor, contributor-mask runs: a mask tile should have about the bytes of a data tile (the stage of the
  // bulk all-gather path holds one), but a unit of A elements is A * mask_bytes >= 16 bytes of masks
  uint32_t mask_tile_units = 0;
  uint64_t mask_tiles_per_rank = 0;
  // column executor: a tile is taken through its list by a whole CTA (0) or by one warp (1), chosen from the plan's
  // shape for the data run and for the contributor-mask run separately
  uint32_t col_warp = 0, mask_warp = 0;
  std::vector<uint64_t> region_offs;    // sorted unique flow offsets (regions tile [0, n), PLAN_SPEC 5.4)
  std::vector<uint64_t> region_len;     // elements of every region
  std::vector<uint32_t> region_flows;   // flows over every region
  std::vector<uint32_t> region_class;   // part * sections + section (P2P pieces: one more class): regions of one class
                                        // differ only in the segment, so their flow lists are the same up to the offset
  std::vector<uint64_t> region_tile0;   // first tile counter of every region (prefix sum)
  optcc_rawvec<uint32_t> flow_region;   // [n_flows] index into region_offs of the region a flow covers
  optcc_exec_state* exec;               // created lazily by the executor; freed by optcc_plan_destroy
};

// implemented in optcc_exec.cu
void optcc_exec_state_free(optcc_exec_state*);
// implemented in optcc_plan.cpp: storage kinds of a bf16 plan in table order (executors that walk the table step by step)
void optcc_assign_kinds(struct optcc_plan*);

// Run body(chunk) for chunk in [0, n) on a few host threads when there is enough work to pay for them; the chunks
// must be independent.
#include <atomic>
#include <thread>
template <class F>
inline void optcc_parallel_chunks(size_t n, size_t work, F body) {
  unsigned hw = std::thread::hardware_concurrency();
  unsigned nt = work < (size_t(1) << 16) ? 1u : std::min(8u, hw ? hw : 1u);
  if (nt <= 1 || n <= 1) { for (size_t i = 0; i < n; ++i) body(i); return; }
  std::atomic<size_t> next{0};
  auto worker = [&]() { for (size_t i; (i = next.fetch_add(1, std::memory_order_relaxed)) < n;) body(i); };
  std::vector<std::thread> th;
  th.reserve(nt - 1);
  for (unsigned t = 1; t < nt; ++t) th.emplace_back(worker);
  worker();
  for (auto& t : th) t.join();
}

// ---- device workspace layout (bytes from the workspace base; every region 256-byte aligned) -----------------
//   control block | rank pointers | device flow records | per-(step, CTA) slice table | dataflow deps, tile-ops | column items | dataflow counters | fp32 shadow (bf16 plans) | masks (verify)
constexpr uint32_t OPTCC_MAX_GRID = 1024;       // upper bound on executor CTAs (sizes the slice table)
constexpr uint64_t OPTCC_CTRL_BYTES = 256;
constexpr uint64_t OPTCC_DFLOW_BYTES = 32;      // sizeof(DFlow) in optcc_exec.cu
constexpr uint64_t OPTCC_SLICE_BYTES = 16;      // sizeof(Slice)

struct optcc_ws_layout {
  uint64_t ctrl, ptrs, dflows, slices, deps, ops, col, col_mask, counters, shadow, masks, end_exec, end_verify;
};

static inline uint64_t optcc_align256(uint64_t x) { return (x + 255) & ~uint64_t(255); }

constexpr uint32_t OPTCC_TILE_UNITS_DEFAULT = 3584;  // largest auto tile: 56 KB of f32 / bf16 = two streaming rounds
constexpr uint64_t OPTCC_DEP_BYTES = 16;             // sizeof(DDep)
constexpr uint64_t OPTCC_OP_BYTES = 8;               // sizeof(TileOp)

static inline optcc_ws_layout optcc_layout(const optcc_plan_t* pl) {
  const optcc_plan_info_t& in = pl->info;
  optcc_ws_layout L;
  L.ctrl = 0;
  L.ptrs = OPTCC_CTRL_BYTES;                                   // rank pointer table (used when p > 128)
  L.dflows = optcc_align256(L.ptrs + uint64_t(in.p) * 8);
  L.slices = optcc_align256(L.dflows + uint64_t(in.n_flows) * OPTCC_DFLOW_BYTES);
  L.deps = optcc_align256(L.slices + uint64_t(in.n_steps) * (OPTCC_MAX_GRID + 1) * OPTCC_SLICE_BYTES);
  L.ops = optcc_align256(L.deps + uint64_t(in.n_flows) * OPTCC_DEP_BYTES);
  L.col = optcc_align256(L.ops + pl->n_tile_ops * OPTCC_OP_BYTES);   // column executor: work items, 16 B per (region, tile)
  L.col_mask = optcc_align256(L.col + pl->tiles_per_rank * 16);      // the verifier's work items when its tiles differ
  L.counters = optcc_align256(L.col_mask + (pl->mask_tile_units != pl->tile_units ? pl->mask_tiles_per_rank * 16 : 0));
  L.shadow = optcc_align256(L.counters + uint64_t(in.p) * pl->tiles_per_rank * 4);
  uint64_t n_pad = (in.n + 7) & ~uint64_t(7);
  L.end_exec = optcc_align256(L.shadow + (in.dtype == OPTCC_BF16 ? uint64_t(in.p) * n_pad * 4 : 0));
  L.masks = L.end_exec;
  L.end_verify = optcc_align256(L.masks + uint64_t(in.p) * n_pad * in.mask_bytes);
  return L;
}

#endif
