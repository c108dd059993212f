// Internal definitions shared by the host planner (optcc_plan.cpp) and the executor (optcc_exec.cu).
// Not part of the ABI.  Nothing here is shared with oracle/ (the oracle is Python and never includes this).
#ifndef OPTCC_INTERNAL_H_
#define OPTCC_INTERNAL_H_

#include <cstdint>
#include <vector>

#include "optcc.h"

// Storage kind of a (rank, region) at some point of a bf16 plan (partial sums stay fp32 between
// steps, one RNE rounding when the sum over all p ranks completes).
enum : uint8_t { OPTCC_KIND_BUF = 0 /* the rank buffer, plan dtype */, OPTCC_KIND_F32 = 1 /* fp32 shadow */ };

struct optcc_exec_state;  // device-side cache, defined in optcc_exec.cu

struct optcc_plan {
  optcc_plan_info_t info;
  optcc_opts_t opts;
  std::vector<double> ell;              // [p]
  std::vector<uint32_t> stragglers;     // server indices, ell descending then index (PLAN_SPEC 1)
  std::vector<uint32_t> healthy;        // server indices ascending
  std::vector<optcc_flow_t> flows;      // sorted (PLAN_SPEC 3)
  std::vector<uint32_t> step_begin;     // [n_steps + 1]
  std::vector<uint64_t> sec_bounds;
  std::vector<uint64_t> p2p_bounds;
  // per flow, bf16 plans only: storage kinds of src, dst before, dst after (host walk over contributor counts)
  std::vector<uint8_t> kind_src, kind_dst_in, kind_dst_out;
  optcc_exec_state* exec;               // created lazily by the executor; freed by optcc_plan_destroy
};

// implemented in optcc_exec.cu
void optcc_exec_state_free(optcc_exec_state*);

// ---- device workspace layout (bytes from the workspace base; every region 256-byte aligned) -----------------
//   control block | rank pointers | device flow records | per-(step, CTA) slice table | fp32 shadow (bf16 plans) | masks (verify)
constexpr uint32_t OPTCC_MAX_GRID = 1024;       // upper bound on executor CTAs (sizes the slice table)
constexpr uint64_t OPTCC_CTRL_BYTES = 256;
constexpr uint64_t OPTCC_DFLOW_BYTES = 32;      // sizeof(DFlow) in optcc_exec.cu
constexpr uint64_t OPTCC_SLICE_BYTES = 16;      // sizeof(Slice)

struct optcc_ws_layout {
  uint64_t ctrl, ptrs, dflows, slices, shadow, masks, end_exec, end_verify;
};

static inline uint64_t optcc_align256(uint64_t x) { return (x + 255) & ~uint64_t(255); }

static inline optcc_ws_layout optcc_layout(const optcc_plan_info_t& in) {
  optcc_ws_layout L;
  L.ctrl = 0;
  L.ptrs = OPTCC_CTRL_BYTES;                                   // rank pointer table (used when p > 128)
  L.dflows = optcc_align256(L.ptrs + uint64_t(in.p) * 8);
  L.slices = optcc_align256(L.dflows + uint64_t(in.n_flows) * OPTCC_DFLOW_BYTES);
  L.shadow = optcc_align256(L.slices + uint64_t(in.n_steps) * (OPTCC_MAX_GRID + 1) * OPTCC_SLICE_BYTES);
  uint64_t n_pad = (in.n + 7) & ~uint64_t(7);
  L.end_exec = optcc_align256(L.shadow + (in.dtype == OPTCC_BF16 ? uint64_t(in.p) * n_pad * 4 : 0));
  L.masks = L.end_exec;
  L.end_verify = optcc_align256(L.masks + uint64_t(in.p) * n_pad * in.mask_words * 8);
  return L;
}

#endif
