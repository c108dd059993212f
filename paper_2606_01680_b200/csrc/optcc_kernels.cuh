// Device code of the OPTCC executor (sm_100a).  Included only by optcc_exec.cu.
//
// Shared device definitions: the device flow / dependency records, the launch parameters and the 16-byte-vector
// range operations every executor uses, for all element types:
//   MODE_F32     rank buffers of float; reduce = one IEEE fp32 add per element ("adds its own section")
//   MODE_BF16    rank buffers of bf16, fp32 partial sums in a shadow array, one RNE rounding when a sum completes (R12)
//   MODE_MASK16 / 32 / 1 / 2   contributor bitmasks of 16 / 32 / 64 / 128 bits: reduce = disjoint OR, copy = assign
// so the verifier (PAPER.md:68 correctness (ii)) runs exactly the tables the executor runs.
//
// Executors (optcc_exec.cu): the column kernels (a tile of one region taken through its whole flow list, CTA-wide or
// warp-wide tiles, no synchronisation between CTAs; the default), the dataflow kernel (tile-ops claimed in table
// order, per-range completion counters, no grid barrier), the persistent kernel (host-built slices of equal HBM bytes
// per step and CTA, grid barrier between steps) and the same kernel launched once per step.  All stream 16-byte
// vectors, fully coalesced, UNROLL independent vectors in flight per thread and stream.
#ifndef OPTCC_KERNELS_CUH_
#define OPTCC_KERNELS_CUH_

#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

namespace optcc_dev {

enum { MODE_F32 = 0, MODE_BF16 = 1, MODE_MASK1 = 2, MODE_MASK2 = 3, MODE_MASK16 = 4, MODE_MASK32 = 5 };
__host__ __device__ constexpr bool is_mask_mode(int m) { return m >= MODE_MASK1; }
// bytes per contributor mask: 16 bits (p <= 16), 32 (p <= 32), 64 (p <= 64), 128 (p <= 128)
__host__ __device__ constexpr int mask_bytes_of(int m) { return m == MODE_MASK16 ? 2 : m == MODE_MASK32 ? 4 : m == MODE_MASK1 ? 8 : 16; }

constexpr int THREADS = 512;      // threads per CTA
constexpr int CTAS_PER_SM = 2;    // resident CTAs per SM the kernels are tuned for (<= 64 registers/thread)
constexpr int STAGE = 16;         // flow records staged in shared memory per CTA and step
constexpr int MAX_PARAM_PTRS = 128;

struct __align__(16) DFlow {      // 32 bytes: what the device needs of an optcc_flow_t
  unsigned long long off;         // elements
  unsigned long long len;         // elements
  unsigned short src, dst;
  unsigned char op, ksrc, kdin, kdout;  // op: 0 reduce, 1 copy; k*: 0 rank buffer, 1 fp32 shadow (bf16 plans)
  unsigned int flags;             // DFLOW_* bits
  unsigned int pad1;
};
static_assert(sizeof(DFlow) == 32, "DFlow must be 32 bytes");
enum : unsigned int {
  DFLOW_DEAD_SRC = 1u,   // the source range is dead after this flow has read it (see discard_line16)
  // first touches and last writes.  Data runs of the column executor request first touches (DRAM accesses) ahead of
  // time; contributor-mask runs in the lazy form (ExecParams.mask_lazy, see range_mask_lazy) take the constant
  // initial mask instead of loading it and let the last writer check the final mask:
  DFLOW_SRC_INIT = 2u,   // no earlier executed flow wrote the source range: it holds rank src's input / the mask {src}
  DFLOW_DST_INIT = 4u,   // no earlier executed flow wrote the destination range (a reduce flow reads it)
  DFLOW_FINAL = 8u,      // no later flow writes the destination range: what this flow writes is the final value / mask
  // column executor, data runs, bulk all-gather path (see build_column_tables / optcc_column_kernel):
  DFLOW_STAGE_OUT = 64u,   // reduce flow: the sum it stores is the source of later copy flows -- also keep it in the CTA's stage
  DFLOW_FROM_STAGE = 128u, // copy flow: the source range holds exactly the staged tile -- store it with cp.async.bulk
  // column executor, one-round tiles (a thread handles the same vectors in every flow of the item): contributor-mask
  // runs in the lazy form (ExecParams.mask_fwd) and data runs (ExecParams.data_fwd bit 1, opts.no_forward = 0):
  DFLOW_SRC_FWD = 256u,    // the source range was written by the previous flow of the list, this flow is its only
                           // reader and the range is overwritten later: the values are taken from the thread's registers
  DFLOW_NO_STORE = 512u,   // ... and that previous flow does not store them (nobody would ever read them from memory;
                           // never set on a final value, on the staged tile or on a copy the bulk path stores)
  // column executor, data runs (ExecParams.data_fwd bit 0):
  DFLOW_SRC_REG = 1024u,   // reduce flow whose source range is what the reduce flow just before it in the list produced:
                           // every thread still holds exactly those vectors in registers and adds them instead of loading
                           // them back through L1 (same bits whether or not that flow stored them)
};

struct __align__(16) Slice {      // start of a CTA's slice of a step: flow index and 16-byte unit inside it
  unsigned int flow;
  unsigned int pad;
  unsigned long long unit;
};
static_assert(sizeof(Slice) == 16, "Slice must be 16 bytes");

struct __align__(16) DDep {       // dataflow dependencies of a flow (same for all its tiles)
  unsigned int csrc, cdst;        // first tile counter of (src rank, region) / (dst rank, region)
  unsigned int need_src;          // accesses of the src range that must be complete before it is read
  unsigned int need_dst;          // accesses of the dst range that must be complete before it is written
};
static_assert(sizeof(DDep) == 16, "DDep must be 16 bytes");

struct TileOp { unsigned int flow, tile; };   // one unit of work of the dataflow executor

constexpr int DF_COMPUTE_THREADS = 448;   // 14 streaming warps
constexpr int DF_SLOTS = 4;               // scheduler agents = tile-ops a CTA can hold (claimed, waiting or streaming)
constexpr int DF_THREADS = DF_COMPUTE_THREADS + 32 * DF_SLOTS;

struct Ctrl {                     // control block at the start of the workspace
  unsigned long long barrier;     // monotone arrival counter of the grid barrier
  unsigned long long bad;         // verify: wrong final masks
  unsigned long long overlap;     // verify: reduce over overlapping contributor sets
  unsigned long long first_bad;   // verify: smallest bad r*n+e
  unsigned long long ticket;      // dataflow: next tile-op to claim
  unsigned long long stamp;       // which plan's tables the workspace holds (written with the tables; see ExecParams.stamp)
  unsigned long long stale;       // launches that found another stamp than theirs and did nothing
};

struct ExecParams {
  void* bufs[MAX_PARAM_PTRS];     // rank buffers (p <= 128); masks: per-rank mask arrays
  void* const* ptr_table;         // rank buffers when p > 128 (device array), else nullptr
  const DFlow* flows;
  const Slice* slices;            // [n_steps][gridDim.x + 1]
  Ctrl* ctrl;
  float* shadow;                  // bf16 plans: fp32 partials, [p][padded_n]
  unsigned long long padded_n;
  unsigned long long n;           // elements per rank (index of a wrong final mask = rank * n + element)
  unsigned int n_ranks;           // p
  unsigned int pad0;
  unsigned int step_lo, step_hi;  // steps [lo, hi) are executed by this launch
  unsigned int unit_elems;        // A (PLAN_SPEC 2)
  unsigned int use_barrier;       // 1: grid barrier between steps (cooperative launch)
  // dataflow executor
  const DDep* deps;               // [n_flows]
  const TileOp* ops;              // [n_ops], table order
  unsigned int* counters;         // [p * tiles_per_rank] completed accesses per (rank, region, tile)
  unsigned long long n_ops;
  unsigned int tile_units;
  unsigned int df_slots;          // ring depth: tile-ops a CTA holds (claimed, waiting or streaming), <= DF_SLOTS
  // column executor: flows are stored region by region (table order inside a region)
  const uint4* col_items;         // [col_n_items] (first flow, end flow of the region in `flows`, tile, units in the tile)
  unsigned long long col_n_items;  // items this launch runs: item i of the launch is entry i * item_stride + item_first of col_items
  unsigned int item_first, item_stride;   // (0, 1) = all items; (s, S) = shard s of S (optcc_execute_shard: peers on other GPUs run the rest)
  unsigned int bulk_copy;         // 1: copy tile-ops are moved by the scheduler agents with cp.async.bulk
  unsigned int l2_hints;          // kind(src loads) + 4 kind(dst loads) + 16 kind(stores); kind: 0 normal, 1 evict_first, 2 evict_last
  unsigned int col_pf_dist;       // column executor: raw operands are requested this many flows ahead (>= 1)
  unsigned int col_pf_l2;         // 1: requested into L2 (prefetch.global.L2), 0: into L1
  unsigned int col_pf_next;       // 1: the look-ahead continues into the CTA's next work item (claimed one item ahead)
  unsigned int col_bulk;          // 1: data runs act on DFLOW_STAGE_OUT / FROM_STAGE (bulk all-gather path)
  unsigned int mask_lazy;         // contributor-mask runs: 1 = lazy form (initial masks are constants, last writers check)
  unsigned int col_bulk_policy;   // L2 policy of the bulk stores (0 normal, 1 evict_first, 2 evict_last)
  unsigned int col_warp;          // 1: warp-wide tiles (optcc_wcolumn_kernel), 0: CTA-wide tiles (optcc_column_kernel)
  unsigned int col_stage_bytes;   // bytes of one staged tile (the warp-wide kernel keeps one per warp)
  unsigned int mask_fwd;          // lazy contributor-mask runs: act on DFLOW_SRC_FWD / DFLOW_NO_STORE
  unsigned int col_chunk;         // warp-wide tiles: 0 = items dealt round-robin to the grid's warps; else a warp claims this many consecutive items at a time
  unsigned int data_fwd;          // data runs, one-round tiles: bit 0 = act on DFLOW_SRC_REG (range_add_f32_round /
                                  // range_add_bf16_round), bit 1 = also on DFLOW_NO_STORE (dead partial sums stay in registers)
  unsigned int pad4;
  unsigned long long stamp;       // the launching plan's table stamp: a kernel whose workspace holds another one (the
                                  // memory was reused, or freed and allocated again at the same address) must not walk
                                  // the tables it finds there -- it counts itself in Ctrl.stale and returns
};

// ---- memory access helpers: L2-only loads (data written by other SMs in the previous step), streaming stores ----
// L2 eviction policies (createpolicy): loads of the streams are evict_first -- a section is dead once the next hop has
// read it, raw destination data is dead once summed -- so that what was just written (the next step's source) stays.
struct Pol { unsigned long long lds, ldd, st; static constexpr unsigned int l1 = 0; };   // source loads, destination loads, stores
struct PolL1 { unsigned long long lds, ldd, st; static constexpr unsigned int l1 = 1; }; // the same, loads and stores through L1
__device__ __forceinline__ unsigned long long make_policy(unsigned int kind) {   // 0 normal, 1 evict_first, 2 evict_last
  unsigned long long p;
  if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// mode = kind(src loads) + 4 * kind(dst loads) + 16 * kind(stores)
__device__ __forceinline__ Pol make_policies(unsigned int mode) {
  Pol p;
  p.lds = make_policy(mode & 3u);
  p.ldd = make_policy((mode >> 2) & 3u);
  p.st = make_policy((mode >> 4) & 3u);
  return p;
}
// l1 = 0: L2 only (.cg) -- the data may have been written by another SM.  l1 = 1 (column executor: a tile is only
// ever touched by the CTA that owns it): default caching, so a value the thread stored one flow earlier is found in L1.
__device__ __forceinline__ uint4 ld16(const void* p, unsigned long long policy, unsigned int l1) {
  uint4 v;
  if (l1)
    asm volatile("ld.global.ca.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(policy) : "memory");
  else
    asm volatile("ld.global.cg.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(policy) : "memory");
  return v;
}
template <class PolX>
__device__ __forceinline__ void st16(void* p, uint4 v, const PolX& pol) {
  if (pol.l1)
    asm volatile("st.global.wb.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;"
                 ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol.st) : "memory");
  else
    asm volatile("st.global.cg.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;"
                 ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol.st) : "memory");
}
__device__ __forceinline__ void sts16(char* smem, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"((unsigned int)__cvta_generic_to_shared(smem)), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ float bf16_to_f32(unsigned int h) { return __uint_as_float(h << 16); }
// float -> bf16 bits, round to nearest even; NaN stays a quiet NaN
__device__ __forceinline__ unsigned int f32_to_bf16_rne(float f) {
  unsigned int u = __float_as_uint(f);
  if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (u >> 16) | 0x40u;
  return (u + 0x7FFFu + ((u >> 16) & 1u)) >> 16;
}

__device__ __forceinline__ uint4 add_f32x4(uint4 a, uint4 b) {
  uint4 r;
  r.x = __float_as_uint(__fadd_rn(__uint_as_float(a.x), __uint_as_float(b.x)));
  r.y = __float_as_uint(__fadd_rn(__uint_as_float(a.y), __uint_as_float(b.y)));
  r.z = __float_as_uint(__fadd_rn(__uint_as_float(a.z), __uint_as_float(b.z)));
  r.w = __float_as_uint(__fadd_rn(__uint_as_float(a.w), __uint_as_float(b.w)));
  return r;
}

// every thread of every kernel starts with this (all threads of the grid take the same branch)
__device__ __forceinline__ bool tables_are_stale(const ExecParams& P) {
  if (__ldcg(&P.ctrl->stamp) == P.stamp) return false;
  if (threadIdx.x == 0 && blockIdx.x == 0) atomicAdd(&P.ctrl->stale, 1ull);
  return true;
}

// ---- grid-wide barrier: every CTA arrives once per step; counter is monotone, target = arrivals expected so far ----
__device__ __forceinline__ void grid_barrier(unsigned long long* ctr, unsigned long long target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long seen;
    asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
    do {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(ctr) : "memory");
    } while (seen < target);
    __threadfence();
  }
  __syncthreads();
}

// =====================================================================================================
// Range operations.  All ranges are given in 16-byte vectors [vbeg, vend) relative to the flow's start.  NT threads
// work on a range together: a whole CTA (thread index = threadIdx.x) or, with NT = 32, one warp on its own
// (thread index = lane) -- the column executor's warps run independent work items.
// =====================================================================================================
template <int NT>
__device__ __forceinline__ unsigned int group_tid() { return NT == 32 ? (threadIdx.x & 31u) : threadIdx.x; }

// Dead-source discard.  When the planner knows that the next access to a flow's source range is a plain overwrite (the
// all-gather copy of the final sum), the data is dead once this flow has read it; dropping its lines from L2
// (discard.global.L2 -> CCTL.RML2) saves the write-back of a partial sum nobody will read again.  A lane discards
// the 128-byte line that starts at its own vector when the line's other vectors were loaded by the following lanes of
// the same warp in the same instruction (so every load of the line has completed before the discard is issued).
__device__ __forceinline__ void discard_line16(const char* addr, unsigned long long v, unsigned long long vend) {
  // 16-byte vectors: a line is 8 consecutive lanes
  if ((reinterpret_cast<unsigned long long>(addr) & 127ull) == 0ull && (threadIdx.x & 31u) <= 24u && v + 7 < vend)
    asm volatile("discard.global.L2 [%0], 128;" ::"l"(addr) : "memory");
}
__device__ __forceinline__ void discard_line32(const char* addr, unsigned long long u, unsigned long long uend) {
  // 32 bytes per lane (fp32 shadow of a bf16 unit): a line is 4 consecutive lanes
  if ((reinterpret_cast<unsigned long long>(addr) & 127ull) == 0ull && (threadIdx.x & 31u) <= 28u && u + 3 < uend)
    asm volatile("discard.global.L2 [%0], 128;" ::"l"(addr) : "memory");
}

// calls f(std::integral_constant<int, rem>) for rem in 1 .. UNROLL-1 (UNROLL <= 8)
template <int UNROLL, class F>
__device__ __forceinline__ void remainder_dispatch(unsigned int rem, F&& f) {
  if (UNROLL > 7 && rem >= 7) f(std::integral_constant<int, 7>());
  else if (UNROLL > 6 && rem == 6) f(std::integral_constant<int, 6>());
  else if (UNROLL > 5 && rem == 5) f(std::integral_constant<int, 5>());
  else if (UNROLL > 4 && rem == 4) f(std::integral_constant<int, 4>());
  else if (UNROLL > 3 && rem >= 3) f(std::integral_constant<int, 3>());
  else if (UNROLL > 2 && rem == 2) f(std::integral_constant<int, 2>());
  else f(std::integral_constant<int, 1>());
}

template <int UNROLL, int NT, class PolX>
__device__ __forceinline__ void range_copy16(const char* __restrict__ s, char* __restrict__ d,
                                             unsigned long long vbeg, unsigned long long vend, const PolX& pol) {
  unsigned long long v = vbeg + group_tid<NT>();
  for (; v + (UNROLL - 1) * (unsigned long long)NT < vend; v += UNROLL * (unsigned long long)NT) {
    uint4 x[UNROLL];
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) x[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) st16(d + (v + j * (unsigned long long)NT) * 16, x[j], pol);
  }
  if (v < vend) {   // remainder (< UNROLL vectors for this thread): still one batch of loads, then the stores
    const unsigned int rem = (unsigned int)((vend - v + NT - 1) / NT);
    auto batch = [&](auto K) {
      constexpr int KK = decltype(K)::value;
      uint4 x[KK];
#pragma unroll
      for (int j = 0; j < KK; ++j) x[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
#pragma unroll
      for (int j = 0; j < KK; ++j) st16(d + (v + j * (unsigned long long)NT) * 16, x[j], pol);
    };
    remainder_dispatch<UNROLL>(rem, batch);
  }
}

// `stage` (column executor, DFLOW_STAGE_OUT): shared-memory image of the tile, vector vbeg at offset 0 -- the sum is
// stored to the destination range as listed and kept in the stage for the bulk all-gather; nullptr otherwise.
template <int UNROLL, int NT, bool STAGE, class PolX>
__device__ __forceinline__ void range_add_f32(const char* __restrict__ s, char* __restrict__ d,
                                              unsigned long long vbeg, unsigned long long vend, const PolX& pol, bool dead_src,
                                              char* stage) {
  unsigned long long v = vbeg + group_tid<NT>();
  for (; v + (UNROLL - 1) * (unsigned long long)NT < vend; v += UNROLL * (unsigned long long)NT) {
    uint4 a[UNROLL], b[UNROLL];
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      a[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
      b[j] = ld16(d + (v + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
    }
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      const uint4 r = add_f32x4(b[j], a[j]);
      st16(d + (v + j * (unsigned long long)NT) * 16, r, pol);
      if (STAGE) sts16(stage + (v + j * (unsigned long long)NT - vbeg) * 16, r);
    }
    // (only when every lane of the warp is in this round: the line's other vectors were loaded by this instruction)
    if (dead_src && (v - (threadIdx.x & 31u) + 31) + (UNROLL - 1) * (unsigned long long)NT < vend) {
#pragma unroll
      for (int j = 0; j < UNROLL; ++j) discard_line16(s + (v + j * (unsigned long long)NT) * 16, v + j * (unsigned long long)NT, vend);
    }
  }
  if (v < vend) {   // remainder: one batch of loads, then the adds and stores
    const unsigned int rem = (unsigned int)((vend - v + NT - 1) / NT);
    auto batch = [&](auto K) {
      constexpr int KK = decltype(K)::value;
      uint4 a[KK], b[KK];
#pragma unroll
      for (int j = 0; j < KK; ++j) {
        a[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
        b[j] = ld16(d + (v + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
      }
#pragma unroll
      for (int j = 0; j < KK; ++j) {
        const uint4 r = add_f32x4(b[j], a[j]);
        st16(d + (v + j * (unsigned long long)NT) * 16, r, pol);
        if (STAGE) sts16(stage + (v + j * (unsigned long long)NT - vbeg) * 16, r);
      }
    };
    remainder_dispatch<UNROLL>(rem, batch);
  }
}

// One round of range_add_f32 with forwarding (ExecParams.data_fwd: the tile is at most one round of four vectors per
// thread, so a thread handles the same vectors in every flow of the item).  `carry` holds the sums this thread stored in
// the previous flow of the list; with src_reg (DFLOW_SRC_REG: that flow's destination is this flow's source) they are
// the source operand -- the load that would return the bits the thread has just stored is not issued.  The add and the
// store to the destination range are issued as listed, so memory holds what the step-ordered executors leave there.
template <int NT, bool STAGE, class PolX>
__device__ __forceinline__ void range_add_f32_round(const char* __restrict__ s, char* __restrict__ d,
                                                    unsigned long long vbeg, unsigned long long vend, const PolX& pol,
                                                    bool dead_src, bool src_reg, char* stage, uint4 (&carry)[4], bool no_store = false) {
  const unsigned long long v0 = vbeg + group_tid<NT>();
  if (v0 >= vend) return;
  auto batch = [&](auto K) {
    constexpr int KK = decltype(K)::value;      // this thread's vectors in the tile: v0 + j NT, j < KK
    uint4 b[KK];
#pragma unroll
    for (int j = 0; j < KK; ++j) b[j] = ld16(d + (v0 + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
    if (!src_reg) {
#pragma unroll
      for (int j = 0; j < KK; ++j) carry[j] = ld16(s + (v0 + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
    }
#pragma unroll
    for (int j = 0; j < KK; ++j) {
      const uint4 r = add_f32x4(b[j], carry[j]);
      carry[j] = r;
      if (!no_store) st16(d + (v0 + j * (unsigned long long)NT) * 16, r, pol);
      if (STAGE) sts16(stage + (v0 + j * (unsigned long long)NT - vbeg) * 16, r);
    }
  };
  if (v0 + 3 * (unsigned long long)NT < vend) {
    batch(std::integral_constant<int, 4>());
    // (only when every lane of the warp is in this round: the line's other vectors are this warp's too)
    if (dead_src && (v0 - (threadIdx.x & 31u) + 31) + 3 * (unsigned long long)NT < vend) {
#pragma unroll
      for (int j = 0; j < 4; ++j) discard_line16(s + (v0 + j * (unsigned long long)NT) * 16, v0 + j * (unsigned long long)NT, vend);
    }
  } else {
    remainder_dispatch<4>((unsigned int)((vend - v0 + NT - 1) / NT), batch);
  }
}

// masks: OR with overlap detection.  EB = bytes per mask element (2, 4, 8 or 16); a 16-byte vector holds 16/EB elements
// stage / all_full (column executor's bulk all-gather path): with `stage`, the joined sets are also kept in that
// shared-memory image of the tile (vector vbeg at offset 0) and all_full is cleared if any of them differs from F
template <int UNROLL, int EB, int NT, class PolX>
__device__ __forceinline__ void range_or_mask(const char* __restrict__ s, char* __restrict__ d,
                                              unsigned long long vbeg, unsigned long long vend,
                                              unsigned int& overlaps, const PolX& pol, bool dead_src,
                                              char* stage = nullptr, uint4 F = make_uint4(0u, 0u, 0u, 0u), bool* all_full = nullptr) {
  auto keep = [&](unsigned long long vv, uint4 o) {
    if (stage) {
      sts16(stage + (vv - vbeg) * 16, o);
      if (((o.x ^ F.x) | (o.y ^ F.y) | (o.z ^ F.z) | (o.w ^ F.w)) != 0u) *all_full = false;
    }
  };
  unsigned long long v = vbeg + group_tid<NT>();
  auto join = [&](uint4 a, uint4 b) {
    const unsigned int cx = a.x & b.x, cy = a.y & b.y, cz = a.z & b.z, cw = a.w & b.w;   // elements whose sets overlap
    if (EB == 2) {
      auto hw = [](unsigned int w) { return ((w & 0xFFFFu) != 0u) + ((w >> 16) != 0u); };
      overlaps += hw(cx) + hw(cy) + hw(cz) + hw(cw);
    } else if (EB == 4) {
      overlaps += (cx != 0u) + (cy != 0u) + (cz != 0u) + (cw != 0u);
    } else if (EB == 8) {
      overlaps += ((cx | cy) != 0u) + ((cz | cw) != 0u);
    } else {
      overlaps += ((cx | cy | cz | cw) != 0u);
    }
    return make_uint4(a.x | b.x, a.y | b.y, a.z | b.z, a.w | b.w);
  };
  for (; v + (UNROLL - 1) * (unsigned long long)NT < vend; v += UNROLL * (unsigned long long)NT) {
    uint4 a[UNROLL], b[UNROLL];
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      a[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
      b[j] = ld16(d + (v + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
    }
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      const uint4 o = join(a[j], b[j]);
      st16(d + (v + j * (unsigned long long)NT) * 16, o, pol);
      keep(v + j * (unsigned long long)NT, o);
    }
    // (only when every lane of the warp is in this round: the line's other vectors were loaded by this instruction)
    if (dead_src && (v - (threadIdx.x & 31u) + 31) + (UNROLL - 1) * (unsigned long long)NT < vend) {
#pragma unroll
      for (int j = 0; j < UNROLL; ++j) discard_line16(s + (v + j * (unsigned long long)NT) * 16, v + j * (unsigned long long)NT, vend);
    }
  }
  if (v < vend) {   // remainder: one batch of loads, then the joins and stores
    const unsigned int rem = (unsigned int)((vend - v + NT - 1) / NT);
    auto batch = [&](auto K) {
      constexpr int KK = decltype(K)::value;
      uint4 a[KK], b[KK];
#pragma unroll
      for (int j = 0; j < KK; ++j) {
        a[j] = ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
        b[j] = ld16(d + (v + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
      }
#pragma unroll
      for (int j = 0; j < KK; ++j) {
        const uint4 o = join(a[j], b[j]);
        st16(d + (v + j * (unsigned long long)NT) * 16, o, pol);
        keep(v + j * (unsigned long long)NT, o);
      }
    };
    remainder_dispatch<UNROLL>(rem, batch);
  }
}

// A 16-byte vector of masks, every element = `bits` (the low EB*8 bits of a 128-bit value given as lo, hi)
__device__ __forceinline__ uint4 mask_vector(unsigned long long lo, unsigned long long hi, unsigned int eb) {
  if (eb == 2) { const unsigned int w = (unsigned int)(lo & 0xFFFFull) * 0x10001u; return make_uint4(w, w, w, w); }
  if (eb == 4) { const unsigned int w = (unsigned int)lo; return make_uint4(w, w, w, w); }
  if (eb == 8) return make_uint4((unsigned int)lo, (unsigned int)(lo >> 32), (unsigned int)lo, (unsigned int)(lo >> 32));
  return make_uint4((unsigned int)lo, (unsigned int)(lo >> 32), (unsigned int)hi, (unsigned int)(hi >> 32));
}

// ---- lazy verifier ----------------------------------------------------------------------------------------------
// The initial mask of rank r is the constant {r}, and the final mask of a range is whatever its last writer stores.
// When the host has seen that every (rank, region) is written by the table (so nothing depends on memory the run
// never wrote), the mask arrays need neither an initialising pass nor a checking pass: a flow whose source /
// destination range has not been written yet takes the constant instead of loading it (DFLOW_SRC_INIT / DST_INIT),
// and the last writer of a range compares what it stores with the full set (DFLOW_FINAL).  Same sets, same stores.

// a wrong final vector (never on a correct plan): count its wrong elements, keep the smallest index
template <int EB>
__device__ __noinline__ void report_bad_masks(unsigned long long* bad_ctr, unsigned long long* first_ctr, uint4 diff,
                                              unsigned long long g) {
  const unsigned int d[4] = {diff.x, diff.y, diff.z, diff.w};
  unsigned long long bad = 0, first = ~0ull;
#pragma unroll
  for (unsigned int j = 0; j < 16 / EB; ++j) {
    bool wrong;
    if (EB == 2) wrong = ((d[j >> 1] >> ((j & 1u) * 16)) & 0xFFFFu) != 0u;
    else if (EB == 4) wrong = d[j] != 0u;
    else if (EB == 8) wrong = (d[2 * j] | d[2 * j + 1]) != 0u;
    else wrong = true;
    if (wrong) { ++bad; if (first == ~0ull) first = g + j; }
  }
  if (bad) {
    atomicAdd(bad_ctr, bad);
    atomicMin(first_ctr, first);
  }
}

// SC / DC: the initial vectors of the source / destination rank, F: the full set; g0 = dst * n + f.off (the global
// index of the flow's first element at its destination); reduce: OR with overlap detection, else assign.
// SRCM: 0 = the source is loaded, 1 = it is the constant SC; DSTM: 0 = copy (no destination operand), 1 = reduce with
// the destination loaded, 2 = reduce with the destination constant DC -- compile-time, so the constants are used in
// place (selecting them at run time cost a register fill per vector).
template <int UNROLL, int EB, int NT, int SRCM, int DSTM, class PolX>
__device__ __forceinline__ void range_mask_lazy_t(const char* __restrict__ s, char* __restrict__ d,
                                                  unsigned long long vbeg, unsigned long long vend, unsigned int& overlaps,
                                                  const PolX& pol, unsigned int flags, uint4 SC, uint4 DC, uint4 F,
                                                  Ctrl* ctrl, unsigned long long g0, char* stage, bool* all_full) {
  constexpr bool src_init = SRCM == 1, dst_init = DSTM == 2, reduce = DSTM != 0;
  const bool fin = (flags & DFLOW_FINAL) != 0u, dead_src = (flags & DFLOW_DEAD_SRC) != 0u && SRCM == 0;
  auto join = [&](uint4 a, uint4 b) {
    const unsigned int cx = a.x & b.x, cy = a.y & b.y, cz = a.z & b.z, cw = a.w & b.w;   // elements whose sets overlap
    if (EB == 2) {
      auto hw = [](unsigned int w) { return ((w & 0xFFFFu) != 0u) + ((w >> 16) != 0u); };
      overlaps += hw(cx) + hw(cy) + hw(cz) + hw(cw);
    } else if (EB == 4) {
      overlaps += (cx != 0u) + (cy != 0u) + (cz != 0u) + (cw != 0u);
    } else if (EB == 8) {
      overlaps += ((cx | cy) != 0u) + ((cz | cw) != 0u);
    } else {
      overlaps += ((cx | cy | cz | cw) != 0u);
    }
    return make_uint4(a.x | b.x, a.y | b.y, a.z | b.z, a.w | b.w);
  };
  const uint4 Z = make_uint4(0u, 0u, 0u, 0u);
  auto batch = [&](unsigned long long v, auto K) {
    constexpr int KK = decltype(K)::value;
    uint4 a[KK], b[KK];
#pragma unroll
    for (int j = 0; j < KK; ++j) {
      a[j] = src_init ? SC : ld16(s + (v + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
      b[j] = !reduce ? Z : (dst_init ? DC : ld16(d + (v + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1));
    }
#pragma unroll
    for (int j = 0; j < KK; ++j) {
      const uint4 o = join(a[j], b[j]);
      st16(d + (v + j * (unsigned long long)NT) * 16, o, pol);
      if (fin || (reduce && stage)) {
        const uint4 df = make_uint4(o.x ^ F.x, o.y ^ F.y, o.z ^ F.z, o.w ^ F.w);
        if ((df.x | df.y | df.z | df.w) != 0u) {
          if (fin) report_bad_masks<EB>(&ctrl->bad, &ctrl->first_bad, df, g0 + (v + j * (unsigned long long)NT) * (16 / EB));
          if (reduce && stage) *all_full = false;
        }
      }
      if (reduce && stage) sts16(stage + (v + j * (unsigned long long)NT - vbeg) * 16, o);
    }
  };
  unsigned long long v = vbeg + group_tid<NT>();
  for (; v + (UNROLL - 1) * (unsigned long long)NT < vend; v += UNROLL * (unsigned long long)NT) {
    batch(v, std::integral_constant<int, UNROLL>());
    // (only when every lane of the warp is in this round: the line's other vectors were loaded by this instruction)
    if (dead_src && (v - (threadIdx.x & 31u) + 31) + (UNROLL - 1) * (unsigned long long)NT < vend) {
#pragma unroll
      for (int j = 0; j < UNROLL; ++j) discard_line16(s + (v + j * (unsigned long long)NT) * 16, v + j * (unsigned long long)NT, vend);
    }
  }
  if (v < vend) {
    const unsigned int rem = (unsigned int)((vend - v + NT - 1) / NT);
    remainder_dispatch<UNROLL>(rem, [&](auto K) { batch(v, K); });
  }
}

// The forwarded ring hop of the verifier, with nothing in memory: carry |= {dst}, overlap detection on the thread's nv
// vectors of the tile (a flow with DFLOW_SRC_FWD, DFLOW_DST_INIT and DFLOW_NO_STORE that is neither final nor staged).
template <int EB>
__device__ __forceinline__ void mask_hop_in_registers(uint4 (&carry)[4], uint4 DC, unsigned int nv, unsigned int& overlaps) {
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint4 a = carry[j];
    const unsigned int cx = a.x & DC.x, cy = a.y & DC.y, cz = a.z & DC.z, cw = a.w & DC.w;
    unsigned int c;
    if (EB == 2) {
      auto hw = [](unsigned int w) { return ((w & 0xFFFFu) != 0u) + ((w >> 16) != 0u); };
      c = hw(cx) + hw(cy) + hw(cz) + hw(cw);
    } else if (EB == 4) {
      c = (cx != 0u) + (cy != 0u) + (cz != 0u) + (cw != 0u);
    } else if (EB == 8) {
      c = ((cx | cy) != 0u) + ((cz | cw) != 0u);
    } else {
      c = ((cx | cy | cz | cw) != 0u);
    }
    if ((unsigned int)j < nv) overlaps += c;
    carry[j] = make_uint4(a.x | DC.x, a.y | DC.y, a.z | DC.z, a.w | DC.w);
  }
}

// One round of the lazy form with forwarding (ExecParams.mask_fwd: the tile is at most one round of UNROLL vectors per
// thread, so a thread handles the same vectors in every flow of the item).  `carry` holds what the previous flow of
// the list produced for them: DFLOW_SRC_FWD takes the source from there instead of loading it, DFLOW_NO_STORE skips the
// store of a result that is only ever read that way and overwritten later.  With both, a ring hop of the verifier is a
// few ALU instructions per vector: the partial sets never travel through L1 / L2.  Flags are warp-uniform.
template <int UNROLL, int EB, int NT, class PolX>
__device__ __forceinline__ void range_mask_round(const char* __restrict__ s, char* __restrict__ d,
                                                 unsigned long long vbeg, unsigned long long vend, unsigned int& overlaps,
                                                 const PolX& pol, unsigned int flags, bool reduce, uint4 SC, uint4 DC, uint4 F,
                                                 Ctrl* ctrl, unsigned long long g0, char* stage, bool* all_full,
                                                 uint4 (&carry)[UNROLL]) {
  const bool src_init = (flags & DFLOW_SRC_INIT) != 0u, src_fwd = (flags & DFLOW_SRC_FWD) != 0u;
  const bool dst_init = (flags & DFLOW_DST_INIT) != 0u, fin = (flags & DFLOW_FINAL) != 0u, ns = (flags & DFLOW_NO_STORE) != 0u;
  const bool dead_src = (flags & DFLOW_DEAD_SRC) != 0u && !src_init && !src_fwd;
  const unsigned long long v0 = vbeg + group_tid<NT>();
  if (v0 >= vend) return;
  auto batch = [&](auto K) {
    constexpr int KK = decltype(K)::value;      // this thread's vectors in the tile: v0 + j NT, j < KK
    uint4 b[KK];
    if (!src_init && !src_fwd) {
#pragma unroll
      for (int j = 0; j < KK; ++j) carry[j] = ld16(s + (v0 + j * (unsigned long long)NT) * 16, pol.lds, pol.l1);
    } else if (src_init) {
#pragma unroll
      for (int j = 0; j < KK; ++j) carry[j] = SC;
    }
    if (reduce && !dst_init) {
#pragma unroll
      for (int j = 0; j < KK; ++j) b[j] = ld16(d + (v0 + j * (unsigned long long)NT) * 16, pol.ldd, pol.l1);
    } else {
      const uint4 c = reduce ? DC : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
      for (int j = 0; j < KK; ++j) b[j] = c;
    }
#pragma unroll
    for (int j = 0; j < KK; ++j) {
      const unsigned long long v = v0 + j * (unsigned long long)NT;
      const uint4 a = carry[j];
      const unsigned int cx = a.x & b[j].x, cy = a.y & b[j].y, cz = a.z & b[j].z, cw = a.w & b[j].w;   // elements whose sets overlap
      if (EB == 2) {
        auto hw = [](unsigned int w) { return ((w & 0xFFFFu) != 0u) + ((w >> 16) != 0u); };
        overlaps += hw(cx) + hw(cy) + hw(cz) + hw(cw);
      } else if (EB == 4) {
        overlaps += (cx != 0u) + (cy != 0u) + (cz != 0u) + (cw != 0u);
      } else if (EB == 8) {
        overlaps += ((cx | cy) != 0u) + ((cz | cw) != 0u);
      } else {
        overlaps += ((cx | cy | cz | cw) != 0u);
      }
      const uint4 o = make_uint4(a.x | b[j].x, a.y | b[j].y, a.z | b[j].z, a.w | b[j].w);
      carry[j] = o;
      if (!ns) st16(d + v * 16, o, pol);
      if (fin || (reduce && stage)) {
        const uint4 df = make_uint4(o.x ^ F.x, o.y ^ F.y, o.z ^ F.z, o.w ^ F.w);
        if ((df.x | df.y | df.z | df.w) != 0u) {
          if (fin) report_bad_masks<EB>(&ctrl->bad, &ctrl->first_bad, df, g0 + v * (16 / EB));
          if (reduce && stage) *all_full = false;
        }
      }
      if (reduce && stage) sts16(stage + (v - vbeg) * 16, o);
    }
  };
  if (v0 + (UNROLL - 1) * (unsigned long long)NT < vend) {
    batch(std::integral_constant<int, UNROLL>());
    // (only when every lane of the warp is in this round: the line's other vectors were loaded by this instruction)
    if (dead_src && (v0 - (threadIdx.x & 31u) + 31) + (UNROLL - 1) * (unsigned long long)NT < vend) {
#pragma unroll
      for (int j = 0; j < UNROLL; ++j) discard_line16(s + (v0 + j * (unsigned long long)NT) * 16, v0 + j * (unsigned long long)NT, vend);
    }
  } else {
    remainder_dispatch<UNROLL>((unsigned int)((vend - v0 + NT - 1) / NT), batch);
  }
}

template <int UNROLL, int EB, int NT, class PolX>
__device__ __forceinline__ void range_mask_lazy(const char* __restrict__ s, char* __restrict__ d,
                                                unsigned long long vbeg, unsigned long long vend, unsigned int& overlaps,
                                                const PolX& pol, unsigned int flags, bool reduce, uint4 SC, uint4 DC, uint4 F,
                                                Ctrl* ctrl, unsigned long long g0, char* stage = nullptr, bool* all_full = nullptr) {
  const int sm = (flags & DFLOW_SRC_INIT) != 0u ? 1 : 0;
  const int dm = !reduce ? 0 : ((flags & DFLOW_DST_INIT) != 0u ? 2 : 1);
#define OPTCC_LAZY_CASE(SM, DM) \
  range_mask_lazy_t<UNROLL, EB, NT, SM, DM>(s, d, vbeg, vend, overlaps, pol, flags, SC, DC, F, ctrl, g0, stage, all_full)
  if (sm == 1) {
    if (dm == 0) OPTCC_LAZY_CASE(1, 0); else if (dm == 1) OPTCC_LAZY_CASE(1, 1); else OPTCC_LAZY_CASE(1, 2);
  } else {
    if (dm == 0) OPTCC_LAZY_CASE(0, 0); else if (dm == 1) OPTCC_LAZY_CASE(0, 1); else OPTCC_LAZY_CASE(0, 2);
  }
#undef OPTCC_LAZY_CASE
}

// A staged tile that is NOT the full set (a wrong or truncated plan) and a copy flow that is the last writer of its
// range: the tile is stored from the stage through the LSU, and every wrong element is reported as the lazy form does.
template <int EB, int NT, class PolX>
__device__ __forceinline__ void range_copy_stage_checked(const char* stage, char* __restrict__ d, unsigned long long vbeg,
                                                         unsigned long long vend, const PolX& pol, uint4 F, Ctrl* ctrl,
                                                         unsigned long long g0) {
  for (unsigned long long v = vbeg + group_tid<NT>(); v < vend; v += NT) {
    uint4 o;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w)
                 : "r"((unsigned int)__cvta_generic_to_shared(stage + (v - vbeg) * 16)) : "memory");
    st16(d + v * 16, o, pol);
    const uint4 df = make_uint4(o.x ^ F.x, o.y ^ F.y, o.z ^ F.z, o.w ^ F.w);
    if ((df.x | df.y | df.z | df.w) != 0u) report_bad_masks<EB>(&ctrl->bad, &ctrl->first_bad, df, g0 + v * (16 / EB));
  }
}

// bf16 plans: a unit is 8 elements = 16 bytes in a rank buffer or 32 bytes in the fp32 shadow.
template <int KIND>
__device__ __forceinline__ void load8(const char* base, unsigned long long unit, float (&x)[8], unsigned long long pol, unsigned int l1) {
  if (KIND == 0) {
    uint4 r = ld16(base + unit * 16, pol, l1);
    x[0] = bf16_to_f32(r.x & 0xFFFFu); x[1] = bf16_to_f32(r.x >> 16);
    x[2] = bf16_to_f32(r.y & 0xFFFFu); x[3] = bf16_to_f32(r.y >> 16);
    x[4] = bf16_to_f32(r.z & 0xFFFFu); x[5] = bf16_to_f32(r.z >> 16);
    x[6] = bf16_to_f32(r.w & 0xFFFFu); x[7] = bf16_to_f32(r.w >> 16);
  } else {
    uint4 r0 = ld16(base + unit * 32, pol, l1), r1 = ld16(base + unit * 32 + 16, pol, l1);
    x[0] = __uint_as_float(r0.x); x[1] = __uint_as_float(r0.y); x[2] = __uint_as_float(r0.z); x[3] = __uint_as_float(r0.w);
    x[4] = __uint_as_float(r1.x); x[5] = __uint_as_float(r1.y); x[6] = __uint_as_float(r1.z); x[7] = __uint_as_float(r1.w);
  }
}
template <int KIND, class PolX>
__device__ __forceinline__ void store8(char* base, unsigned long long unit, const float (&x)[8], const PolX& pol) {
  if (KIND == 0) {
    uint4 r;
    r.x = f32_to_bf16_rne(x[0]) | (f32_to_bf16_rne(x[1]) << 16);
    r.y = f32_to_bf16_rne(x[2]) | (f32_to_bf16_rne(x[3]) << 16);
    r.z = f32_to_bf16_rne(x[4]) | (f32_to_bf16_rne(x[5]) << 16);
    r.w = f32_to_bf16_rne(x[6]) | (f32_to_bf16_rne(x[7]) << 16);
    st16(base + unit * 16, r, pol);
  } else {
    st16(base + unit * 32, make_uint4(__float_as_uint(x[0]), __float_as_uint(x[1]), __float_as_uint(x[2]), __float_as_uint(x[3])), pol);
    st16(base + unit * 32 + 16, make_uint4(__float_as_uint(x[4]), __float_as_uint(x[5]), __float_as_uint(x[6]), __float_as_uint(x[7])), pol);
  }
}

// bf16 image of 8 sums for the stage (the same rounding store8<0> applies)
__device__ __forceinline__ uint4 pack8_bf16(const float (&x)[8]) {
  uint4 r;
  r.x = f32_to_bf16_rne(x[0]) | (f32_to_bf16_rne(x[1]) << 16);
  r.y = f32_to_bf16_rne(x[2]) | (f32_to_bf16_rne(x[3]) << 16);
  r.z = f32_to_bf16_rne(x[4]) | (f32_to_bf16_rne(x[5]) << 16);
  r.w = f32_to_bf16_rne(x[6]) | (f32_to_bf16_rne(x[7]) << 16);
  return r;
}

// `stage`: as in range_add_f32 (only with KO == 0: complete sums live in the rank buffer), one 16-byte unit per slot
template <int KS, int KD, int KO, int NT, class PolX>
__device__ __forceinline__ void range_add_bf16(const char* __restrict__ s, const char* __restrict__ din,
                                               char* __restrict__ dout, unsigned long long ubeg,
                                               unsigned long long uend, const PolX& pol, bool dead_src, char* stage) {
  constexpr int UNROLL = 2;
  unsigned long long u = ubeg + group_tid<NT>();
  for (; u + (UNROLL - 1) * (unsigned long long)NT < uend; u += UNROLL * (unsigned long long)NT) {
    float a[UNROLL][8], b[UNROLL][8];
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      load8<KS>(s, u + j * (unsigned long long)NT, a[j], pol.lds, pol.l1);
      load8<KD>(din, u + j * (unsigned long long)NT, b[j], pol.ldd, pol.l1);
    }
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
#pragma unroll
      for (int e = 0; e < 8; ++e) b[j][e] = __fadd_rn(b[j][e], a[j][e]);
      store8<KO>(dout, u + j * (unsigned long long)NT, b[j], pol);
      if (KO == 0 && stage) sts16(stage + (u + j * (unsigned long long)NT - ubeg) * 16, pack8_bf16(b[j]));
    }
    if (dead_src && (u - (threadIdx.x & 31u) + 31) + (UNROLL - 1) * (unsigned long long)NT < uend) {
#pragma unroll
      for (int j = 0; j < UNROLL; ++j) {
        const unsigned long long uu = u + j * (unsigned long long)NT;
        if (KS == 0) discard_line16(s + uu * 16, uu, uend); else discard_line32(s + uu * 32, uu, uend);
      }
    }
  }
  for (; u < uend; u += NT) {
    float a[8], b[8];
    load8<KS>(s, u, a, pol.lds, pol.l1);
    load8<KD>(din, u, b, pol.ldd, pol.l1);
#pragma unroll
    for (int e = 0; e < 8; ++e) b[e] = __fadd_rn(b[e], a[e]);
    store8<KO>(dout, u, b, pol);
    if (KO == 0 && stage) sts16(stage + (u - ubeg) * 16, pack8_bf16(b));
  }
}

// One round of range_add_bf16 with forwarding (ExecParams.data_fwd: the tile is at most one round of U units per thread).
// `carry` holds, as 8 fp32 values per unit (two uint4), what this thread produced in the previous flow of the list:
// with src_reg (DFLOW_SRC_REG) that is the source operand.  no_store (DFLOW_NO_STORE, fp32 partials only): the result is
// read by the next flow from `carry` alone and its range is overwritten later, so the partial sum is not written to the
// library's fp32 scratch at all.  Rank buffers see exactly the stores range_add_bf16 issues.
// (the KK units of one thread: u0 + j NT, j < KK)
template <int KS, int KD, int KO, int NT, int KK, int CN, class PolX>
__device__ __forceinline__ void bf16_round_batch(const char* __restrict__ s, const char* __restrict__ din, char* __restrict__ dout,
                                                 unsigned long long ubeg, unsigned long long u0, const PolX& pol, bool src_reg,
                                                 bool no_store, char* stage, uint4 (&carry)[CN]) {
  constexpr int W = KD ? 2 : 1;               // the destination operand stays packed until its unit is added
  uint4 braw[KK][W];
#pragma unroll
  for (int j = 0; j < KK; ++j) {
    const char* q = din + (u0 + j * (unsigned long long)NT) * (KD ? 32 : 16);
    braw[j][0] = ld16(q, pol.ldd, pol.l1);
    if (KD) braw[j][W - 1] = ld16(q + 16, pol.ldd, pol.l1);
  }
  if (!src_reg) {
#pragma unroll
    for (int j = 0; j < KK; ++j) {
      const char* q = s + (u0 + j * (unsigned long long)NT) * (KS ? 32 : 16);
      const uint4 r0 = ld16(q, pol.lds, pol.l1);
      if (KS) {
        carry[2 * j] = r0;
        carry[2 * j + 1] = ld16(q + 16, pol.lds, pol.l1);
      } else {
        carry[2 * j] = make_uint4(r0.x << 16, r0.x & 0xFFFF0000u, r0.y << 16, r0.y & 0xFFFF0000u);
        carry[2 * j + 1] = make_uint4(r0.z << 16, r0.z & 0xFFFF0000u, r0.w << 16, r0.w & 0xFFFF0000u);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < KK; ++j) {
    float b[8];
    if (KD) {
      b[0] = __uint_as_float(braw[j][0].x); b[1] = __uint_as_float(braw[j][0].y); b[2] = __uint_as_float(braw[j][0].z); b[3] = __uint_as_float(braw[j][0].w);
      b[4] = __uint_as_float(braw[j][W - 1].x); b[5] = __uint_as_float(braw[j][W - 1].y); b[6] = __uint_as_float(braw[j][W - 1].z); b[7] = __uint_as_float(braw[j][W - 1].w);
    } else {
      const uint4 r = braw[j][0];
      b[0] = bf16_to_f32(r.x & 0xFFFFu); b[1] = bf16_to_f32(r.x >> 16); b[2] = bf16_to_f32(r.y & 0xFFFFu); b[3] = bf16_to_f32(r.y >> 16);
      b[4] = bf16_to_f32(r.z & 0xFFFFu); b[5] = bf16_to_f32(r.z >> 16); b[6] = bf16_to_f32(r.w & 0xFFFFu); b[7] = bf16_to_f32(r.w >> 16);
    }
    const uint4 c0 = carry[2 * j], c1 = carry[2 * j + 1];
    b[0] = __fadd_rn(b[0], __uint_as_float(c0.x)); b[1] = __fadd_rn(b[1], __uint_as_float(c0.y));
    b[2] = __fadd_rn(b[2], __uint_as_float(c0.z)); b[3] = __fadd_rn(b[3], __uint_as_float(c0.w));
    b[4] = __fadd_rn(b[4], __uint_as_float(c1.x)); b[5] = __fadd_rn(b[5], __uint_as_float(c1.y));
    b[6] = __fadd_rn(b[6], __uint_as_float(c1.z)); b[7] = __fadd_rn(b[7], __uint_as_float(c1.w));
    if (KO == 0) {   // the complete sum is rounded when it is stored: `carry` holds what a load of it would return
#pragma unroll
      for (int e = 0; e < 8; ++e) b[e] = bf16_to_f32(f32_to_bf16_rne(b[e]));
    }
    carry[2 * j] = make_uint4(__float_as_uint(b[0]), __float_as_uint(b[1]), __float_as_uint(b[2]), __float_as_uint(b[3]));
    carry[2 * j + 1] = make_uint4(__float_as_uint(b[4]), __float_as_uint(b[5]), __float_as_uint(b[6]), __float_as_uint(b[7]));
    if (!no_store) store8<KO>(dout, u0 + j * (unsigned long long)NT, b, pol);
    if (KO == 0 && stage) sts16(stage + (u0 + j * (unsigned long long)NT - ubeg) * 16, pack8_bf16(b));
  }
}

template <int KS, int KD, int KO, int NT, int U, class PolX>
__device__ __forceinline__ void range_add_bf16_round(const char* __restrict__ s, const char* __restrict__ din,
                                                     char* __restrict__ dout, unsigned long long ubeg, unsigned long long uend,
                                                     const PolX& pol, bool dead_src, bool src_reg, bool no_store, char* stage,
                                                     uint4 (&carry)[2 * U]) {
  const unsigned long long u0 = ubeg + group_tid<NT>();
  if (u0 >= uend) return;
  if (u0 + (U - 1) * (unsigned long long)NT < uend) {
    bf16_round_batch<KS, KD, KO, NT, U>(s, din, dout, ubeg, u0, pol, src_reg, no_store, stage, carry);
    if (dead_src && (u0 - (threadIdx.x & 31u) + 31) + (U - 1) * (unsigned long long)NT < uend) {
#pragma unroll
      for (int j = 0; j < U; ++j) {
        const unsigned long long uu = u0 + j * (unsigned long long)NT;
        if (KS == 0) discard_line16(s + uu * 16, uu, uend); else discard_line32(s + uu * 32, uu, uend);
      }
    }
  } else {
    const unsigned int rem = (unsigned int)((uend - u0 + NT - 1) / NT);
    if (U > 3 && rem >= 3) bf16_round_batch<KS, KD, KO, NT, (U > 3 ? 3 : 1)>(s, din, dout, ubeg, u0, pol, src_reg, no_store, stage, carry);
    else if (U > 2 && rem == 2) bf16_round_batch<KS, KD, KO, NT, (U > 2 ? 2 : 1)>(s, din, dout, ubeg, u0, pol, src_reg, no_store, stage, carry);
    else bf16_round_batch<KS, KD, KO, NT, 1>(s, din, dout, ubeg, u0, pol, src_reg, no_store, stage, carry);
  }
}

}  // namespace optcc_dev
#endif
