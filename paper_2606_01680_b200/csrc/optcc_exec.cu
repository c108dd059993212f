// Executor and verifier of liboptcc (sm_100a): carries out an OPTCC plan over p virtual ranks' buffers held in one
// GPU's HBM.  Reduce flows (Stage 1 hops PAPER.md:126, Stage 3 fold-in :132, bubble-up :165, NVLink collect :862-875)
// are range additions dst[R] += src[R]; copy flows (Stage 4 :136, Stage 2 :130, bubble-down :165, NVLink distribute
// :863-876) are range copies.  Four executors run the same tables and give the same bits: two keep the global step
// order (persistent kernel with a grid barrier; one launch per step), the dataflow kernel orders tile-ops by per-range
// completion counters, and the column kernels (the default) take a tile of one region through every flow over that
// region in an order that respects the data dependencies of :138 inside the element column -- every flow's add is
// carried out in the plan's order, a partial sum that only the next flow of the column reads and a later flow
// overwrites stays in registers, and there is no global step order.  The verifier runs the same tables on
// contributor bitmasks.  No tensor cores: nothing here is a dense contraction.
#include <algorithm>
#include <cstring>
#include <new>
#include <atomic>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "optcc_internal.h"
#include "optcc_kernels.cuh"

using namespace optcc_dev;

static_assert(sizeof(DFlow) == OPTCC_DFLOW_BYTES, "layout constant out of date");
static_assert(sizeof(Slice) == OPTCC_SLICE_BYTES, "layout constant out of date");
static_assert(sizeof(Ctrl) <= OPTCC_CTRL_BYTES, "control block too large");

namespace {

thread_local int g_last_cuda_error = 0;

#define CU_TRY(call)                          \
  do {                                        \
    cudaError_t e_ = (call);                  \
    if (e_ != cudaSuccess) {                  \
      g_last_cuda_error = (int)e_;            \
      (void)cudaGetLastError();               \
      return OPTCC_ECUDA;                     \
    }                                         \
  } while (0)

template <int MODE> struct ModeTraits;
template <> struct ModeTraits<MODE_F32>   { static constexpr int ESIZE = 4,  VE = 4; };
template <> struct ModeTraits<MODE_BF16>  { static constexpr int ESIZE = 2,  VE = 8; };
template <> struct ModeTraits<MODE_MASK1> { static constexpr int ESIZE = 8,  VE = 2; };
template <> struct ModeTraits<MODE_MASK2> { static constexpr int ESIZE = 16, VE = 1; };
template <> struct ModeTraits<MODE_MASK16> { static constexpr int ESIZE = 2, VE = 8; };
template <> struct ModeTraits<MODE_MASK32> { static constexpr int ESIZE = 4, VE = 4; };

__device__ __forceinline__ char* rank_ptr(const ExecParams& P, unsigned int r) {
  return reinterpret_cast<char*>(P.ptr_table ? P.ptr_table[r] : P.bufs[r]);
}

// One piece of one flow: 16-byte units [ubeg, uend) of the flow, executed by the whole CTA.
// stage / from_stage (column executor's bulk all-gather path, data runs): a reduce flow with `stage` also keeps the sum
// it stores in that shared-memory image of the tile; a copy flow with `from_stage` has its whole vectors stored by one
// thread's cp.async.bulk (see optcc_column_kernel), only the ragged end of a buffer is moved here.
// carry / use_carry (lazy contributor-mask runs of the column executor): the sets this thread produced in the previous
// flow of the list, taken instead of a load when the flow says so (DFLOW_SRC_FWD); other callers pass a scratch array.
// MASK_FWD (column executor, contributor-mask runs): the run is in the lazy form and every tile is one round, so only
// the forwarding round (range_mask_round) is compiled in -- the kernel then has the registers to keep `carry` live.
// MASK_FWD with MODE_F32 (column executor, ExecParams.data_fwd): every tile is one round, reduce flows run as
// range_add_f32_round and take a source the previous flow stored (DFLOW_SRC_REG) from `carry` instead of loading it.
template <int MODE, int NT, bool MASK_FWD = false, class PolX, int CN>
__device__ __forceinline__ void process_piece(const ExecParams& P, const DFlow& f, unsigned long long ubeg,
                                              unsigned long long uend, unsigned int& overlaps, const PolX& pol,
                                              uint4 (&carry)[CN], bool use_carry = false,
                                              char* stage = nullptr, bool from_stage = false, bool* stage_full = nullptr) {
  using MT = ModeTraits<MODE>;
  const unsigned int tid = group_tid<NT>();
  const unsigned long long A = P.unit_elems;
  const unsigned long long e0 = ubeg * A;
  unsigned long long e1 = uend * A;
  if (e1 > f.len) e1 = f.len;
  if (e0 >= e1) return;
  const bool dead_src = (f.flags & 1u) != 0u;
  const unsigned long long vbeg = e0 / MT::VE, vend = e1 / MT::VE;  // full 16-byte vectors
  const unsigned int tail = (unsigned int)(e1 % MT::VE);            // ragged end of the buffer (n not a multiple of A)

  if (MODE == MODE_F32) {
    const char* s = rank_ptr(P, f.src) + f.off * 4;
    char* d = rank_ptr(P, f.dst) + f.off * 4;
    if (f.op == 0 && MASK_FWD) {   // (data runs: FWD = ExecParams.data_fwd, the tile is one round)
      const bool src_reg = use_carry && (f.flags & DFLOW_SRC_REG) != 0u;
      const bool elide = (P.data_fwd & 2u) != 0u;
      const bool no_store = elide && (f.flags & DFLOW_NO_STORE) != 0u;
      const bool dead = dead_src && !(elide && (f.flags & DFLOW_SRC_FWD));   // (a source that was never stored has no dirty line)
      uint4 (&c4)[4] = reinterpret_cast<uint4 (&)[4]>(carry);
      if (stage) range_add_f32_round<NT, true>(s, d, vbeg, vend, pol, dead, src_reg, stage, c4, no_store);
      else range_add_f32_round<NT, false>(s, d, vbeg, vend, pol, dead, src_reg, nullptr, c4, no_store);
    } else if (f.op == 0) {
      if (stage) range_add_f32<4, NT, true>(s, d, vbeg, vend, pol, dead_src, stage);
      else range_add_f32<4, NT, false>(s, d, vbeg, vend, pol, dead_src, nullptr);
    } else if (!from_stage) {
      range_copy16<4, NT>(s, d, vbeg, vend, pol);
    }
    if (tid < tail) {
      unsigned long long e = vend * 4 + tid;
      const float* sf = reinterpret_cast<const float*>(s);
      float* df = reinterpret_cast<float*>(d);
      float x = __ldcg(sf + e);
      if (f.op == 0) x = __fadd_rn(__ldcg(df + e), x);
      __stcg(df + e, x);
    }
  } else if (is_mask_mode(MODE)) {
    constexpr int EB = MT::ESIZE;
    const char* s = rank_ptr(P, f.src) + f.off * EB;
    char* d = rank_ptr(P, f.dst) + f.off * EB;
    const unsigned int lazy = P.mask_lazy ? f.flags & (DFLOW_SRC_INIT | DFLOW_DST_INIT | DFLOW_FINAL) : 0u;
    const unsigned long long full0 = P.n_ranks >= 64 ? ~0ull : ((1ull << P.n_ranks) - 1ull);
    const unsigned long long full1 = P.n_ranks > 64 ? (P.n_ranks >= 128 ? ~0ull : ((1ull << (P.n_ranks - 64)) - 1ull)) : 0ull;
    if (from_stage) {
      // whole vectors: stored by cp.async.bulk from the stage -- or, when this copy is the last writer of its range
      // (lazy form) and the staged sets are not all complete, through the LSU with every wrong element reported
      if (stage)
        range_copy_stage_checked<EB, NT>(stage, d, vbeg, vend, pol, mask_vector(full0, full1, EB), P.ctrl,
                                         (unsigned long long)f.dst * P.n + f.off);
    } else if (MASK_FWD) {      // lazy form, one round per tile: partial sets are forwarded through `carry`
      const uint4 SC = mask_vector(f.src < 64 ? 1ull << f.src : 0ull, f.src >= 64 ? 1ull << (f.src - 64) : 0ull, EB);
      const uint4 DC = mask_vector(f.dst < 64 ? 1ull << f.dst : 0ull, f.dst >= 64 ? 1ull << (f.dst - 64) : 0ull, EB);
      range_mask_round<4, EB, NT>(s, d, vbeg, vend, overlaps, pol, f.flags, f.op == 0, SC, DC, mask_vector(full0, full1, EB),
                                  P.ctrl, (unsigned long long)f.dst * P.n + f.off, f.op == 0 ? stage : nullptr, stage_full,
                                  reinterpret_cast<uint4 (&)[4]>(carry));
    } else if (P.mask_lazy) {   // lazy verifier: initial masks are constants, the last writer checks the final mask (range_mask_lazy)
      const uint4 SC = mask_vector(f.src < 64 ? 1ull << f.src : 0ull, f.src >= 64 ? 1ull << (f.src - 64) : 0ull, EB);
      const uint4 DC = mask_vector(f.dst < 64 ? 1ull << f.dst : 0ull, f.dst >= 64 ? 1ull << (f.dst - 64) : 0ull, EB);
      range_mask_lazy<4, EB, NT>(s, d, vbeg, vend, overlaps, pol, f.flags, f.op == 0, SC, DC, mask_vector(full0, full1, EB),
                                 P.ctrl, (unsigned long long)f.dst * P.n + f.off, f.op == 0 ? stage : nullptr, stage_full);
    } else if (f.op == 0) {
      range_or_mask<4, EB, NT>(s, d, vbeg, vend, overlaps, pol, dead_src, stage, mask_vector(full0, full1, EB), stage_full);
    } else {
      range_copy16<4, NT>(s, d, vbeg, vend, pol);
    }
    if (tid < tail) {  // ragged end (n not a multiple of the elements per vector): one element per thread
      const unsigned long long e = vend * MT::VE + tid;   // (EB <= 8 here: a 16-byte mask is a whole vector)
      unsigned long long x, y = 0;
      if (lazy & DFLOW_SRC_INIT) {
        x = 1ull << f.src;
      } else if (EB == 2) {
        x = __ldcg(reinterpret_cast<const unsigned short*>(s) + e);
      } else if (EB == 4) {
        x = __ldcg(reinterpret_cast<const unsigned int*>(s) + e);
      } else {
        x = __ldcg(reinterpret_cast<const unsigned long long*>(s) + e);
      }
      if (f.op == 0) {
        if (lazy & DFLOW_DST_INIT) y = 1ull << f.dst;
        else if (EB == 2) y = __ldcg(reinterpret_cast<const unsigned short*>(d) + e);
        else if (EB == 4) y = __ldcg(reinterpret_cast<const unsigned int*>(d) + e);
        else y = __ldcg(reinterpret_cast<const unsigned long long*>(d) + e);
      }
      overlaps += (x & y) != 0ull;
      x |= y;
      if ((lazy & DFLOW_FINAL) && x != full0) {
        atomicAdd(&P.ctrl->bad, 1ull);
        atomicMin(&P.ctrl->first_bad, (unsigned long long)f.dst * P.n + f.off + e);
      }
      if (EB == 2) __stcg(reinterpret_cast<unsigned short*>(d) + e, (unsigned short)x);
      else if (EB == 4) __stcg(reinterpret_cast<unsigned int*>(d) + e, (unsigned int)x);
      else __stcg(reinterpret_cast<unsigned long long*>(d) + e, x);
    }
  } else {  // MODE_BF16
    const char* s = f.ksrc ? reinterpret_cast<const char*>(P.shadow + (unsigned long long)f.src * P.padded_n + f.off)
                           : rank_ptr(P, f.src) + f.off * 2;
    const char* di = f.kdin ? reinterpret_cast<const char*>(P.shadow + (unsigned long long)f.dst * P.padded_n + f.off)
                            : rank_ptr(P, f.dst) + f.off * 2;
    char* dout = f.kdout ? reinterpret_cast<char*>(P.shadow + (unsigned long long)f.dst * P.padded_n + f.off)
                         : rank_ptr(P, f.dst) + f.off * 2;
    if (f.op == 0) {
      // (dead-source discard is off for bf16 plans in the dataflow executor: measured 3 % slower on C3, which is not
      // DRAM-bound there; on in the column executor)
      const bool bf_dead = PolX::l1 != 0 && dead_src;
      if (MASK_FWD) {   // (data runs: FWD = ExecParams.data_fwd, the tile is one round of CN / 2 units per thread)
        constexpr int U = CN / 2;
        const bool src_reg = use_carry && (f.flags & DFLOW_SRC_REG) != 0u;
        const bool elide = (P.data_fwd & 2u) != 0u;
        const bool ns = elide && (f.flags & DFLOW_NO_STORE) != 0u;
        const bool dd = bf_dead && !(elide && (f.flags & DFLOW_SRC_FWD));
        switch ((f.ksrc << 2) | (f.kdin << 1) | f.kdout) {
          case 0: range_add_bf16_round<0, 0, 0, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 1: range_add_bf16_round<0, 0, 1, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 2: range_add_bf16_round<0, 1, 0, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 3: range_add_bf16_round<0, 1, 1, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 4: range_add_bf16_round<1, 0, 0, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 5: range_add_bf16_round<1, 0, 1, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          case 6: range_add_bf16_round<1, 1, 0, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
          default: range_add_bf16_round<1, 1, 1, NT, U>(s, di, dout, vbeg, vend, pol, dd, src_reg, ns, stage, carry); break;
        }
      } else
      switch ((f.ksrc << 2) | (f.kdin << 1) | f.kdout) {
        case 0: range_add_bf16<0, 0, 0, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 1: range_add_bf16<0, 0, 1, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 2: range_add_bf16<0, 1, 0, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 3: range_add_bf16<0, 1, 1, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 4: range_add_bf16<1, 0, 0, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 5: range_add_bf16<1, 0, 1, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        case 6: range_add_bf16<1, 1, 0, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
        default: range_add_bf16<1, 1, 1, NT>(s, di, dout, vbeg, vend, pol, bf_dead, stage); break;
      }
    } else if (from_stage) {
      // (whole units stored by cp.async.bulk from the stage)
    } else if (f.ksrc == 0) {
      range_copy16<4, NT>(s, dout, vbeg, vend, pol);                 // bf16 -> bf16: one vector per unit
    } else {
      range_copy16<4, NT>(s, dout, vbeg * 2, vend * 2, pol);         // fp32 partial -> fp32 partial: two vectors per unit
    }
    if (tid < tail) {
      unsigned long long e = vend * 8 + tid;
      float x = f.ksrc ? __ldcg(reinterpret_cast<const float*>(s) + e)
                       : bf16_to_f32(__ldcg(reinterpret_cast<const unsigned short*>(s) + e));
      if (f.op == 0) {
        float y = f.kdin ? __ldcg(reinterpret_cast<const float*>(di) + e)
                         : bf16_to_f32(__ldcg(reinterpret_cast<const unsigned short*>(di) + e));
        x = __fadd_rn(y, x);
      }
      if (f.kdout) __stcg(reinterpret_cast<float*>(dout) + e, x);
      else __stcg(reinterpret_cast<unsigned short*>(dout) + e, (unsigned short)f32_to_bf16_rne(x));
    }
  }
}

// The executor kernel.  gridDim.x CTAs; CTA c executes slice c of every step in [step_lo, step_hi).
template <int MODE>
__global__ void __launch_bounds__(THREADS, CTAS_PER_SM) optcc_exec_kernel(const __grid_constant__ ExecParams P) {
  if (tables_are_stale(P)) return;
  __shared__ DFlow s_flow[2][STAGE];             // the CTA's part of the step table, staged one step ahead
  __shared__ unsigned long long s_ubeg[2], s_uend[2];
  __shared__ unsigned int s_f0[2], s_nf[2];

  const unsigned int G = gridDim.x, cta = blockIdx.x;
  unsigned int overlaps = 0;
  uint4 scratch[4];
  const Pol pol = make_policies(P.l2_hints);

  auto stage = [&](unsigned int step, int buf, unsigned int lane) {
    // called by one warp: fetch the slice bounds and up to STAGE flow records of `step`
    const Slice* sl = P.slices + (unsigned long long)step * (G + 1) + cta;
    const uint4 ra = __ldg(reinterpret_cast<const uint4*>(sl)), rb = __ldg(reinterpret_cast<const uint4*>(sl + 1));
    const unsigned int a_flow = ra.x, b_flow = rb.x;
    const unsigned long long a_unit = ra.z | ((unsigned long long)ra.w << 32), b_unit = rb.z | ((unsigned long long)rb.w << 32);
    unsigned int nf = b_flow - a_flow + (b_unit > 0 ? 1u : 0u);
    if (lane == 0) { s_f0[buf] = a_flow; s_nf[buf] = nf; s_ubeg[buf] = a_unit; s_uend[buf] = b_unit; }
    if (lane < nf && lane < STAGE) {
      const uint4* src = reinterpret_cast<const uint4*>(P.flows + a_flow + lane);
      uint4* dst = reinterpret_cast<uint4*>(&s_flow[buf][lane]);
      dst[0] = __ldg(src);
      dst[1] = __ldg(src + 1);
    }
  };

  if (threadIdx.x < 32) stage(P.step_lo, P.step_lo & 1, threadIdx.x);
  __syncthreads();

  for (unsigned int step = P.step_lo; step < P.step_hi; ++step) {
    const int buf = step & 1;
    if (step + 1 < P.step_hi && threadIdx.x >= THREADS - 32) stage(step + 1, buf ^ 1, threadIdx.x - (THREADS - 32));
    const unsigned int f0 = s_f0[buf], nf = s_nf[buf];
    const unsigned long long ub = s_ubeg[buf], ue = s_uend[buf];
    for (unsigned int i = 0; i < nf; ++i) {
      DFlow f;
      if (i < STAGE) {
        f = s_flow[buf][i];
      } else {  // more flows in one slice than staged: read the record from the table directly
        const uint4* src = reinterpret_cast<const uint4*>(P.flows + f0 + i);
        uint4 lo = __ldg(src), hi = __ldg(src + 1);
        memcpy(&f, &lo, 16);
        memcpy(reinterpret_cast<char*>(&f) + 16, &hi, 16);
      }
      const unsigned long long A = P.unit_elems;
      const unsigned long long nunits = (f.len + A - 1) / A;
      const unsigned long long ubeg = i == 0 ? ub : 0ull;
      const unsigned long long uend = (i + 1 == nf && ue > 0) ? ue : nunits;
      process_piece<MODE, THREADS>(P, f, ubeg, uend, overlaps, pol, scratch);
    }
    if (step + 1 < P.step_hi) {
      if (P.use_barrier) grid_barrier(&P.ctrl->barrier, (unsigned long long)(step - P.step_lo + 1) * G);
      else __syncthreads();
    }
  }

  if (is_mask_mode(MODE)) {
    // warp-shuffle reduction of the per-thread overlap counts, one atomic per warp
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) overlaps += __shfl_xor_sync(0xFFFFFFFFu, overlaps, o);
    if ((threadIdx.x & 31) == 0 && overlaps) atomicAdd(&P.ctrl->overlap, (unsigned long long)overlaps);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Dataflow executor: no grid barrier.  14 streaming warps + up to 4 scheduler agents (one lane each) per CTA.
// Agent w owns slot w of a small ring in shared memory (this CTA's staged part of the segment table): it claims the
// next tile-op (global ticket, table order; claims are made in turn), fetches its flow record into the slot, waits
// until the accesses the op depends on have completed (per-(rank, region, tile) counters, ld.acquire.gpu), puts the
// slot into the CTA's ready queue, waits for the streaming warps to finish it, then fences and bumps the counters of
// the two ranges the op touched.  Streaming warps never synchronise with each other: each takes the next entry of the
// ready queue, streams its share and bumps a shared done-counter.  An op only waits on ops with smaller tickets, each
// held by a resident CTA (cooperative launch), and streaming warps only see ops whose dependencies are satisfied --
// progress is guaranteed.
// ---------------------------------------------------------------------------------------------------------
// ---- cp.async.bulk (TMA 1-D bulk copy) helpers for the all-gather (copy) tile-ops -----------------------------
constexpr unsigned int BULK_CHUNK = 4096;     // bytes per bulk transfer
constexpr unsigned int BULK_STAGES = 4;       // chunks in flight per scheduler agent
constexpr unsigned int BULK_SMEM_PER_AGENT = BULK_CHUNK * BULK_STAGES;

__device__ __forceinline__ unsigned int smem_u32(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned int parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_LOOP_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@!p bra WAIT_LOOP_%=;\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, unsigned int bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, unsigned int bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(void* gdst, const void* smem_src, unsigned int bytes, unsigned long long policy) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes), "l"(policy) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// byte extent of units [ubeg, uend) of a copy flow in the current element mode
template <int MODE>
__device__ __forceinline__ void copy_extent(const ExecParams& P, const DFlow& f, unsigned long long ubeg,
                                            unsigned long long uend, const char** src, char** dst,
                                            unsigned long long* nbytes) {
  const unsigned long long A = P.unit_elems, e0 = ubeg * A;
  unsigned long long e1 = uend * A;
  if (e1 > f.len) e1 = f.len;
  unsigned long long esz;
  const char* s;
  char* d;
  if (MODE == MODE_F32) {
    esz = 4; s = rank_ptr(P, f.src); d = rank_ptr(P, f.dst);
  } else if (is_mask_mode(MODE)) {
    esz = mask_bytes_of(MODE); s = rank_ptr(P, f.src); d = rank_ptr(P, f.dst);
  } else if (f.ksrc == 0) {
    esz = 2; s = rank_ptr(P, f.src); d = rank_ptr(P, f.dst);
  } else {
    esz = 4;
    s = reinterpret_cast<const char*>(P.shadow + (unsigned long long)f.src * P.padded_n);
    d = reinterpret_cast<char*>(P.shadow + (unsigned long long)f.dst * P.padded_n);
  }
  *src = s + (f.off + e0) * esz;
  *dst = d + (f.off + e0) * esz;
  *nbytes = e1 > e0 ? (e1 - e0) * esz : 0;
}

// One thread copies nbytes (src, dst 16-byte aligned) global -> shared -> global with bulk async copies, as a
// continuous pipeline over a ring of BULK_STAGES chunks: chunk c is stored as soon as it has landed and its stage is
// reloaded with chunk c + BULK_STAGES once the store has read it, so BULK_STAGES - 1 loads stay in flight.
// `parity` holds one phase bit per stage barrier.
__device__ __forceinline__ void bulk_copy(char* stage, unsigned long long* bars, unsigned int& parity,
                                          const char* src, char* dst, unsigned long long nbytes) {
  const unsigned long long n16 = nbytes & ~15ull;
  const unsigned long long nch = (n16 + BULK_CHUNK - 1) / BULK_CHUNK;
  auto chunk_bytes = [&](unsigned long long c) {
    const unsigned long long o = c * BULK_CHUNK;
    return (unsigned int)(n16 - o < BULK_CHUNK ? n16 - o : BULK_CHUNK);
  };
  auto load = [&](unsigned long long c) {
    const unsigned int st = (unsigned int)(c % BULK_STAGES), b = chunk_bytes(c);
    mbar_expect_tx(bars + st, b);
    bulk_g2s(stage + st * BULK_CHUNK, src + c * BULK_CHUNK, b, bars + st);
  };
  for (unsigned long long c = 0; c < nch && c < BULK_STAGES; ++c) load(c);
  for (unsigned long long c = 0; c < nch; ++c) {
    const unsigned int st = (unsigned int)(c % BULK_STAGES);
    mbar_wait(bars + st, (parity >> st) & 1u);
    parity ^= 1u << st;
    bulk_s2g(dst + c * BULK_CHUNK, stage + st * BULK_CHUNK, chunk_bytes(c));
    if (c + BULK_STAGES < nch) {
      bulk_wait_read_all();        // the store has read its stage: reload it
      load(c + BULK_STAGES);
    }
  }
  bulk_wait_all();                 // every store has been performed
  for (unsigned long long o = n16; o < nbytes; ++o) dst[o] = src[o];   // ragged end of a buffer (< 16 bytes)
}

struct DfSlot {
  DFlow f;
  unsigned long long ubeg, uend;
  unsigned int valid;
  unsigned int pad[3];
};

__device__ __forceinline__ unsigned int ld_acquire_gpu_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned int ld_acquire_cta_shared_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"((unsigned int)__cvta_generic_to_shared(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_cta_shared_u32(unsigned int* p, unsigned int v) {
  asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"((unsigned int)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_cta_shared_add(unsigned int* p, unsigned int v) {
  asm volatile("red.release.cta.shared.add.u32 [%0], %1;" ::"r"((unsigned int)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}

template <int MODE>
__global__ void __launch_bounds__(DF_THREADS, CTAS_PER_SM) optcc_dataflow_kernel(const __grid_constant__ ExecParams P) {
  if (tables_are_stale(P)) return;
  constexpr unsigned int NW = DF_COMPUTE_THREADS / 32;   // streaming warps
  const unsigned int NS = P.df_slots;                    // slots in the ring = scheduler agents in use (<= DF_SLOTS)
  __shared__ DfSlot s_slot[DF_SLOTS];
  constexpr unsigned int QN = 2 * DF_SLOTS;   // ready queue: slots in the order their dependencies were satisfied
  __shared__ unsigned int s_queue[QN];        // entry q % QN: slot number, or QSTOP
  __shared__ unsigned int s_qflag[QN];        // entry q % QN is valid when the flag reads q + 1
  __shared__ unsigned int s_tail;             // next queue position
  __shared__ unsigned int s_exhausted;        // agents that found no ticket left
  constexpr unsigned int QSTOP = 0xFFFFFFFFu;
  __shared__ unsigned int s_done[DF_SLOTS];   // streaming warps that finished ops of the slot (monotone)
  __shared__ unsigned int s_turn;             // local sequence number whose ticket is claimed next
  __shared__ __align__(8) unsigned long long s_bar[DF_SLOTS][BULK_STAGES];   // mbarriers of the bulk-copy stages
  extern __shared__ __align__(128) char s_stage[];   // bulk-copy staging: BULK_SMEM_PER_AGENT per agent (copy_path 2)
  if (threadIdx.x < DF_SLOTS) s_done[threadIdx.x] = 0;
  if (threadIdx.x < QN) s_qflag[threadIdx.x] = 0;
  if (threadIdx.x == 0) {
    s_turn = 0;
    s_tail = 0;
    s_exhausted = 0;
    for (unsigned int a = 0; a < DF_SLOTS; ++a)
      for (unsigned int c = 0; c < BULK_STAGES; ++c) mbar_init(&s_bar[a][c], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  unsigned int overlaps = 0;
  const Pol pol = make_policies(P.l2_hints);

  if (threadIdx.x >= DF_COMPUTE_THREADS) {
    // ---------------- scheduler agents: warp w (lane 0) owns slot w and the ops j = w, w + NS, ... ----------------
    const unsigned int w = (threadIdx.x - DF_COMPUTE_THREADS) >> 5;
    if ((threadIdx.x & 31) != 0 || w >= NS) return;
    DfSlot& sl = s_slot[w];
    unsigned int bulk_parity = 0;
    // state of the op streaming from my slot (cur) and of the op fetched ahead into registers (nxt)
    unsigned int* cur_src = nullptr; unsigned int* cur_dst = nullptr;
    unsigned int cur_target = 0;
    bool cur_pending = false;                    // queued, not yet completed
    auto try_complete = [&]() {                  // every streaming warp is done with cur -> publish its writes
      if (cur_pending && ld_acquire_cta_shared_u32(&s_done[w]) >= cur_target) {
        __threadfence();
        atomicAdd(cur_src, 1u);
        atomicAdd(cur_dst, 1u);
        cur_pending = false;
      }
    };
    for (unsigned int j = w;; j += NS) {
      // ---- claim and fetch op j (while the previous op of this slot may still be streaming) ----
      // tickets are claimed in turn, so that inside a CTA the local order is the table order
      while (ld_acquire_cta_shared_u32(&s_turn) != j) try_complete();
      const unsigned long long t = atomicAdd(&P.ctrl->ticket, 1ull);
      st_release_cta_shared_u32(&s_turn, j + 1);
      try_complete();
      const bool valid = t < P.n_ops;
      unsigned long long opw = 0;
      if (valid) opw = __ldg(reinterpret_cast<const unsigned long long*>(P.ops + t));
      try_complete();
      const unsigned int flow = (unsigned int)opw, tile = (unsigned int)(opw >> 32);
      uint4 f0 = make_uint4(0, 0, 0, 0), f1 = f0, dp = f0;
      if (valid) {
        const uint4* fr = reinterpret_cast<const uint4*>(P.flows + flow);
        f0 = __ldg(fr); f1 = __ldg(fr + 1);
        dp = __ldg(reinterpret_cast<const uint4*>(P.deps + flow));
      }
      // ---- the slot must be free before it is refilled ----
      while (cur_pending) try_complete();
      if (!valid) {                    // nothing left; the last agent to get here queues the stop marker
        if (atomicAdd(&s_exhausted, 1u) == NS - 1) {
          const unsigned int pos = atomicAdd(&s_tail, 1u);
          s_queue[pos % QN] = QSTOP;
          st_release_cta_shared_u32(&s_qflag[pos % QN], pos + 1);
        }
        return;
      }
      memcpy(&sl.f, &f0, 16);
      memcpy(reinterpret_cast<char*>(&sl.f) + 16, &f1, 16);
      const unsigned long long A = P.unit_elems, nunits = (sl.f.len + A - 1) / A;
      sl.ubeg = (unsigned long long)tile * P.tile_units;
      sl.uend = sl.ubeg + P.tile_units < nunits ? sl.ubeg + P.tile_units : nunits;
      const bool bulk = P.bulk_copy && sl.f.op == 1;   // all-gather tile-op: this agent moves it with cp.async.bulk
      sl.valid = bulk ? 2 : 1;
      cur_src = P.counters + dp.x + tile;
      cur_dst = P.counters + dp.y + tile;
      // the accesses this op depends on (PAPER.md:138 data dependencies), per (rank, region, tile)
      // (a range nobody has touched yet needs no look at its counter: raw inputs, first writes)
      if (dp.z) while (ld_acquire_gpu_u32(cur_src) < dp.z) { }
      if (dp.w) while (ld_acquire_gpu_u32(cur_dst) < dp.w) { }
      {   // ready: queue the slot.  The streaming warps take slots in readiness order, so an op that still waits
          // for its dependencies never holds up a later one that is ready.
        const unsigned int pos = atomicAdd(&s_tail, 1u);
        s_queue[pos % QN] = w;
        st_release_cta_shared_u32(&s_qflag[pos % QN], pos + 1);
      }
      cur_target = NW * (j / NS + 1);
      cur_pending = true;
      if (bulk) {
        const char* src;
        char* dst;
        unsigned long long nbytes;
        copy_extent<MODE>(P, sl.f, sl.ubeg, sl.uend, &src, &dst, &nbytes);
        fence_proxy_async();   // the source was written through the generic proxy by other CTAs
        bulk_copy(s_stage + w * BULK_SMEM_PER_AGENT, s_bar[w], bulk_parity, src, dst, nbytes);
        fence_proxy_async();
      }
      // completion happens inside the next iteration's claim / fetch (try_complete), overlapped with it
    }
  } else {
    // ---------------- streaming warps ----------------
    for (unsigned int q = 0;; ++q) {
      while (ld_acquire_cta_shared_u32(&s_qflag[q % QN]) != q + 1) { }
      const unsigned int s = s_queue[q % QN];
      if (s == QSTOP) break;
      const unsigned int kind = s_slot[s].valid;
      if (kind == 1) {   // kind 2: the agent copies it with cp.async.bulk; the streaming warps move on
        const DFlow f = s_slot[s].f;
        const unsigned long long ubeg = s_slot[s].ubeg, uend = s_slot[s].uend;
        uint4 scratch[4];
        process_piece<MODE, DF_COMPUTE_THREADS>(P, f, ubeg, uend, overlaps, pol, scratch);
      }
      __syncwarp();
      if ((threadIdx.x & 31) == 0) red_release_cta_shared_add(&s_done[s], 1u);
    }
    if (is_mask_mode(MODE)) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) overlaps += __shfl_xor_sync(0xFFFFFFFFu, overlaps, o);
      if ((threadIdx.x & 31) == 0 && overlaps) atomicAdd(&P.ctrl->overlap, (unsigned long long)overlaps);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// Column executor: no synchronisation between CTAs.  A flow moves a range from one rank to another at the same
// offset, so no flow mixes two element indices and every data dependency of :138 lies inside one
// element column.  A work item is one tile of one region; the CTA that claims it runs every flow over that region
// on the tile, in table order (the flow records are stored region by region).  Thread i handles the same vectors of
// the tile in every flow, so the ordering a dependent flow needs is the thread's own program order: each flow still
// loads its operands from and stores its result to memory (L2) as listed -- nothing is carried in registers -- and
// the tile's p ranks stay in L2 from the first hop to the last.
// ---------------------------------------------------------------------------------------------------------
constexpr int COL_THREADS = DF_COMPUTE_THREADS;

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// First touches ahead of time.  The ranges of flow f that no earlier flow of the region has written (DFLOW_SRC_INIT /
// DFLOW_DST_INIT, a walk of the table on the host: a ring hop's destination is the next rank's untouched section, the
// straggler's raw section, a raw P2P piece) are DRAM accesses; they are requested col_pf_dist flows before f runs.
// Every thread asks for the vectors it will load itself (NT-strided, like the range operations).  f32 and bf16 data
// only (raw data always lives in the rank buffer): the verifier's first touches are constants.
template <int MODE, int NT>
__device__ __forceinline__ void prefetch_raw(const ExecParams& P, const DFlow& f, unsigned long long ubeg, unsigned int n) {
  if (is_mask_mode(MODE)) return;
  const unsigned int esz = MODE == MODE_F32 ? 4 : 2;
  auto span = [&](const char* base) {
    const char* q = base + (ubeg + group_tid<NT>()) * 16;
    if (P.col_pf_l2) { for (unsigned int u = group_tid<NT>(); u < n; u += NT, q += NT * 16) prefetch_l2(q); }
    else { for (unsigned int u = group_tid<NT>(); u < n; u += NT, q += NT * 16) prefetch_l1(q); }
  };
  if (f.flags & DFLOW_SRC_INIT) span(rank_ptr(P, f.src) + f.off * esz);
  if (f.op == 0 && (f.flags & DFLOW_DST_INIT)) span(rank_ptr(P, f.dst) + f.off * esz);
}

constexpr unsigned int COL_REC = 256;   // flow records staged in shared memory at a time (8 KB)
constexpr unsigned int COL_PF_MAX = 8;  // deepest look-ahead (flows)

template <int MODE, bool MASK_FWD = false>
__global__ void __launch_bounds__(COL_THREADS, CTAS_PER_SM) optcc_column_kernel(const __grid_constant__ ExecParams P) {
  if (tables_are_stale(P)) return;
  __shared__ unsigned long long s_item[2];          // work items are claimed one item ahead
  __shared__ __align__(16) DFlow s_rec[COL_REC];    // this CTA's staged part of the region's flow list
  __shared__ __align__(16) DFlow s_nrec[COL_PF_MAX];   // the first records of the next item (look-ahead across items)
  unsigned int overlaps = 0;
  // A tile is private to its CTA for the whole launch, so loads and stores go through L1 (PolL1): the value a flow
  // stores is the next flow's source.  L2 policies all evict_normal (a dirty line marked evict_first is written back).
  const Pol pol0 = make_policies(P.l2_hints);
  PolL1 pol;
  pol.lds = pol0.lds; pol.ldd = pol0.ldd; pol.st = pol0.st;
  const unsigned int D = is_mask_mode(MODE) ? 0u : (P.col_pf_dist < COL_PF_MAX ? P.col_pf_dist : COL_PF_MAX);
  extern __shared__ __align__(128) char s_stage_col[];   // bulk all-gather path: the tile of the sum being distributed
  const bool bulk = P.col_bulk != 0;
  bool stage_ok = true;              // contributor masks: every staged set is the full set
  unsigned int bulk_turn = 0;        // bulk stores issued so far (the warps' first lanes take turns)
  uint4 carry[4];                    // lazy contributor-mask runs: what the previous flow produced (DFLOW_SRC_FWD)
  const unsigned long long bulk_pol = make_policy(P.col_bulk_policy);   // L2 policy of the bulk stores
  // The first two items of every CTA are dealt statically, the ticket hands out the rest (counting from 2 gridDim.x):
  // same-address atomics from 148 SMs complete about one per 90 ns, and 2 x 296 of them at the start of the kernel kept
  // the last CTA waiting for 50 us (all of C1's kernel time).
  const unsigned long long ticket0 = 2ull * gridDim.x;
  unsigned long long it = blockIdx.x, nit = (unsigned long long)blockIdx.x + gridDim.x;
  bool prefetched = false;           // the first flows of this item were requested during the previous item
  for (unsigned int round = 0; it < P.col_n_items; ++round) {
    // one record per item: the region's flows [fb, fe), the tile and its length in units (all flows over a region have
    // the same length, PLAN_SPEC 5.4, so the tile's unit range is fixed for the item)
    const uint4 item = __ldg(P.col_items + (it * P.item_stride + P.item_first));
    const unsigned int fb = item.x, fe = item.y;
    const unsigned long long ubeg = (unsigned long long)item.z * P.tile_units;
    const unsigned long long uend = ubeg + item.w;
    // look-ahead into the next item: its first raw operands are requested while this item's last flows run
    unsigned long long n_ubeg = 0;
    unsigned int n_cnt = 0, n_units = 0, n_fb = 0;
    if (D && P.col_pf_next && nit < P.col_n_items) {
      const uint4 ni = __ldg(P.col_items + (nit * P.item_stride + P.item_first));
      n_fb = ni.x;
      n_cnt = ni.y - ni.x < D ? ni.y - ni.x : D;
      n_ubeg = (unsigned long long)ni.z * P.tile_units;
      n_units = ni.w;
    }
    int prev_cls = -1;
    // the tile in bytes of the run's element type (all flows over a region have the region's offset and length)
    bool ragged = false;
    unsigned long long tile_byte0 = 0;
    unsigned int tile_bytes = 0, nv = 0;
    for (unsigned int base = fb; base < fe; base += COL_REC) {
      const unsigned int cnt = fe - base < COL_REC ? fe - base : COL_REC;
      const bool last_chunk = base + cnt == fe;
      if (base != fb) __syncthreads();             // the previous records have been read by every thread
      for (unsigned int t = threadIdx.x; t < 2 * cnt; t += COL_THREADS)
        reinterpret_cast<uint4*>(s_rec)[t] = __ldg(reinterpret_cast<const uint4*>(P.flows + base) + t);
      if (base == fb && threadIdx.x < 2 * n_cnt)
        reinterpret_cast<uint4*>(s_nrec)[threadIdx.x] = __ldg(reinterpret_cast<const uint4*>(P.flows + n_fb) + threadIdx.x);
      __syncthreads();
      if (base == fb && D && !prefetched)          // nobody has asked for the first flows' operands yet
        for (unsigned int j = 0; j < D && j < cnt; ++j) prefetch_raw<MODE, COL_THREADS>(P, s_rec[j], ubeg, item.w);
      if (base == fb) {
        constexpr unsigned long long ESZ = ModeTraits<MODE>::ESIZE, VE = 16 / ESZ;
        const unsigned long long len = s_rec[0].len, e0 = ubeg * P.unit_elems;
        unsigned long long e1 = uend * P.unit_elems;
        ragged = e1 > len && (len % VE) != 0;
        if (e1 > len) e1 = len;
        const unsigned long long v0 = e0 / VE, v1 = e1 / VE;     // whole 16-byte vectors of the tile
        tile_byte0 = v0 * 16;
        tile_bytes = (unsigned int)((v1 - v0) * 16);
        const unsigned long long mine0 = v0 + threadIdx.x;
        nv = mine0 >= v1 ? 0u : (unsigned int)((v1 - mine0 + COL_THREADS - 1) / COL_THREADS);
      }
      auto run_flow = [&](const DFlow& cur) {
        if (MODE == MODE_BF16) {
          // a copy of fp32 partials moves two vectors per unit, thread i taking vector i instead of unit i: when the
          // thread-to-element mapping changes between consecutive flows the CTA synchronises (block-wide ordering)
          const int cls = (cur.op == 1 && cur.ksrc != 0) ? 1 : 0;
          if (prev_cls >= 0 && cls != prev_cls) __syncthreads();
          prev_cls = cls;
        }
        // Fast paths (the verifier is bound by instruction issue, ncu r02: 69-72 % of the issue slots): flows that touch
        // no memory from this thread skip everything else.  `ragged`: the tile holds the ragged end of a buffer, whose
        // last few elements always go through memory (process_piece's scalar tail).
        if (MASK_FWD && is_mask_mode(MODE) && !ragged && cur.op == 0 &&
            (cur.flags & (DFLOW_SRC_FWD | DFLOW_DST_INIT | DFLOW_NO_STORE | DFLOW_FINAL | DFLOW_STAGE_OUT)) ==
                (DFLOW_SRC_FWD | DFLOW_DST_INIT | DFLOW_NO_STORE)) {
          constexpr int EB = ModeTraits<MODE>::ESIZE;
          mask_hop_in_registers<EB>(reinterpret_cast<uint4 (&)[4]>(carry), mask_vector(cur.dst < 64 ? 1ull << cur.dst : 0ull, cur.dst >= 64 ? 1ull << (cur.dst - 64) : 0ull, EB),
                                    nv, overlaps);
          return;
        }
        if (bulk && !ragged && (cur.flags & DFLOW_FROM_STAGE) &&
            !(is_mask_mode(MODE) && P.mask_lazy && (cur.flags & DFLOW_FINAL) && !stage_ok)) {
          // the copies of one tile are issued by the warps' first lanes in turn: 60+ cp.async.bulk per tile (C3: every
          // section goes to p - 1 ranks) would otherwise queue behind one thread
          if (threadIdx.x == (bulk_turn % (COL_THREADS / 32)) * 32)
            bulk_s2g_hint(rank_ptr(P, cur.dst) + cur.off * ModeTraits<MODE>::ESIZE + tile_byte0, s_stage_col, tile_bytes, bulk_pol);
          ++bulk_turn;
          return;
        }
        if (bulk) {
          // Bulk all-gather path.  The reduce flow that completes a sum which later copy flows distribute
          // (DFLOW_STAGE_OUT, found by the host's walk of the region's list) stores it to its destination as listed
          // and also keeps it in shared memory; every copy flow whose source range holds exactly that tile
          // (DFLOW_FROM_STAGE) is then one cp.async.bulk store of the staged tile to its destination, issued by one
          // thread in list order -- the all-gather steps move through the TMA unit instead of LDG / STG.
          // Contributor masks, lazy form: a copy that is the last writer of its range must check what it stores; the
          // staged sets are checked once (stage_ok), and only if they are not all complete (a wrong or truncated
          // plan) such copies go through the LSU and report every wrong element.
          const unsigned int fl = cur.flags;
          if (fl & DFLOW_STAGE_OUT) {        // the stage is rewritten: the previous tile's bulk stores must have read it
            if ((threadIdx.x & 31u) == 0) bulk_wait_read_all();   // (every warp's first lane issues bulk stores, in turn)
            __syncthreads();
            bool mine = true;
            process_piece<MODE, COL_THREADS, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, true, s_stage_col, false, &mine);
            // this thread's generic-proxy writes (the stage; its earlier stores to ranges the bulk stores will overwrite)
            // are ordered before the async-proxy operations issued after the barrier
            fence_proxy_async();
            if (is_mask_mode(MODE)) stage_ok = __syncthreads_and(mine) != 0; else __syncthreads();
          } else if (fl & DFLOW_FROM_STAGE) {
            if (is_mask_mode(MODE) && P.mask_lazy && (fl & DFLOW_FINAL) && !stage_ok) {
              process_piece<MODE, COL_THREADS, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, false, s_stage_col, true);
            } else {
              // the copies of one tile are issued by the warps' first lanes in turn: 60+ cp.async.bulk per tile (C3: every
              // section goes to p - 1 ranks) would otherwise queue behind one thread
              if (threadIdx.x == (bulk_turn % (COL_THREADS / 32)) * 32) {
                constexpr unsigned long long ESZ = ModeTraits<MODE>::ESIZE, VE = 16 / ESZ;
                const unsigned long long e0 = ubeg * P.unit_elems;
                unsigned long long e1 = uend * P.unit_elems;
                if (e1 > cur.len) e1 = cur.len;
                const unsigned long long v0 = e0 / VE, v1 = e1 / VE;
                if (v1 > v0) bulk_s2g_hint(rank_ptr(P, cur.dst) + cur.off * ESZ + v0 * 16, s_stage_col, (unsigned int)((v1 - v0) * 16), bulk_pol);
              }
              ++bulk_turn;
              process_piece<MODE, COL_THREADS, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, false, nullptr, true);   // (ragged end of a buffer only)
            }
          } else {
            process_piece<MODE, COL_THREADS, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, true);
          }
        } else {
          process_piece<MODE, COL_THREADS, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, true);
        }
        __syncwarp();   // orders a lane's dead-source discard of a 128-byte line before the other lanes' later stores to it
      };
      if (is_mask_mode(MODE)) {
        // the verifier is bound by instruction issue (ncu: 79 % of the issue slots): records are read in place
        for (unsigned int j = 0; j < cnt; ++j) run_flow(s_rec[j]);
      } else {
        // data: the next record is in registers before its flow starts (its loads issue without waiting for shared memory)
        DFlow cur = s_rec[0];
        for (unsigned int j = 0; j < cnt; ++j) {
          // the raw operands of the flow D places ahead are requested while this one streams (prefetches are hints: a
          // request that is skipped at a chunk boundary or for a very short list costs time, never correctness)
          if (j + D < cnt) prefetch_raw<MODE, COL_THREADS>(P, s_rec[j + D], ubeg, item.w);
          else if (last_chunk && j + D - cnt < n_cnt) prefetch_raw<MODE, COL_THREADS>(P, s_nrec[j + D - cnt], n_ubeg, n_units);
          const DFlow nxt = s_rec[j + 1 < cnt ? j + 1 : j];
          run_flow(cur);
          cur = nxt;
        }
      }
    }
    if (threadIdx.x == 0) s_item[round & 1] = ticket0 + atomicAdd(&P.ctrl->ticket, 1ull);   // (slot of `it`: read by everyone long ago)
    __syncthreads();                 // every thread has read this item's records
    prefetched = n_cnt != 0;
    it = nit;
    nit = s_item[round & 1];
  }
  if (bulk && (threadIdx.x & 31u) == 0) bulk_wait_all();   // the stage stays valid until every bulk store has read it
  __syncthreads();                   // (shared memory is released when the last thread leaves)
  if (is_mask_mode(MODE)) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) overlaps += __shfl_xor_sync(0xFFFFFFFFu, overlaps, o);
    if ((threadIdx.x & 31) == 0 && overlaps) atomicAdd(&P.ctrl->overlap, (unsigned long long)overlaps);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Column executor, warp-wide tiles: the same work items, but one WARP takes a tile (128 units = 4 vectors per lane for
// f32) through its region's list, and the warps of a CTA never wait for each other: no block barrier anywhere, so a
// warp whose loads miss does not hold up thirteen others at the next barrier (the CTA-wide kernel spends a third of its
// stall time there), short regions (C4 at large k: 273 units) keep every warp busy, and items are claimed per warp.
// Records are read straight from the table (uniform loads, L1 hits after the first warp).  Everything else -- table
// order per element, every flow's add carried out, partial sums forwarded in registers, first touches requested one flow ahead, dead-source
// discard, the bulk all-gather path with one stage per warp -- is as in optcc_column_kernel.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ DFlow load_record(const DFlow* p) {
  const uint4 lo = __ldg(reinterpret_cast<const uint4*>(p)), hi = __ldg(reinterpret_cast<const uint4*>(p) + 1);
  DFlow f;
  memcpy(&f, &lo, 16);
  memcpy(reinterpret_cast<char*>(&f) + 16, &hi, 16);
  return f;
}

// A FULL warp-wide tile of an fp32 plan with forwarding (128 units, four vectors per lane, no ragged end) through its
// region's records [fb, fe): the same flows, flags and arithmetic as the generic path (process_piece /
// range_add_f32_round), written as the tight loop a stand-alone probe of this access pattern runs at 0.96 of the copy
// peak with: only the second half of a record is read (src, dst, op, flags -- offset and length are the
// region's), a lane's byte offset is formed once per item, and a flow is its loads, adds and stores.  Measured against
// the generic path in the same run: C4 0.91 vs 1.06 ms, C4 at k = 8 0.95 vs 1.00, C2 on warp-wide tiles 1.43 vs 1.54.
// tile_off: bytes from the start of a rank buffer to the tile; v0 / vend: the lane's first vector and the tile's end
// in the region's vectors (the discard's whole-line test).
template <class PolX>
__device__ __forceinline__ void lean_item_f32(const ExecParams& P, unsigned int fb, unsigned int fe, unsigned long long tile_off,
                                              unsigned int lane, char* stage, const PolX& pol, unsigned long long bulk_pol,
                                              unsigned long long v0, unsigned long long vend, uint4 (&acc)[4]) {
  const bool elide = (P.data_fwd & 2u) != 0u, bulk = P.col_bulk != 0u, pf = P.col_pf_dist != 0u;
  const unsigned long long lane_off = tile_off + lane * 16ull;
  const uint4* const rec = reinterpret_cast<const uint4*>(P.flows + fb) + 1;     // second 16 bytes of record fb
  uint4 cur = __ldg(rec);
  auto first_touches = [&](const uint4& r) {     // the raw operands of a flow are DRAM accesses: requested a flow ahead
    if (r.z & DFLOW_SRC_INIT) { const char* q = rank_ptr(P, r.x & 0xFFFFu) + lane_off; for (int k = 0; k < 4; ++k) prefetch_l1(q + k * 512); }
    if ((r.y & 0xFFu) == 0u && (r.z & DFLOW_DST_INIT)) { const char* q = rank_ptr(P, r.x >> 16) + lane_off; for (int k = 0; k < 4; ++k) prefetch_l1(q + k * 512); }
  };
  if (pf) first_touches(cur);
  for (unsigned int j = fb; j < fe; ++j) {
    const uint4 nxt = __ldg(rec + 2 * ((j + 1 < fe ? j + 1 : j) - fb));
    const unsigned int src = cur.x & 0xFFFFu, dst = cur.x >> 16, fl = cur.z;
    if (pf && j + 1 < fe) first_touches(nxt);
    if ((cur.y & 0xFFu) != 0u) {       // copy
      if (bulk && (fl & DFLOW_FROM_STAGE)) {
        if (lane == 0) bulk_s2g_hint(rank_ptr(P, dst) + tile_off, stage, 128u * 16u, bulk_pol);
      } else {
        const char* sp = rank_ptr(P, src) + lane_off;
        char* dp = rank_ptr(P, dst) + lane_off;
        uint4 x[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) x[k] = ld16(sp + k * 512, pol.lds, pol.l1);
#pragma unroll
        for (int k = 0; k < 4; ++k) st16(dp + k * 512, x[k], pol);
        __syncwarp();
      }
    } else {                           // reduce: dst += src, one IEEE add per element
      char* dp = rank_ptr(P, dst) + lane_off;
      const char* sp = rank_ptr(P, src) + lane_off;
      uint4 b[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) b[k] = ld16(dp + k * 512, pol.ldd, pol.l1);
      if (!(fl & DFLOW_SRC_REG)) {
#pragma unroll
        for (int k = 0; k < 4; ++k) acc[k] = ld16(sp + k * 512, pol.lds, pol.l1);
      }
      const bool staged = bulk && (fl & DFLOW_STAGE_OUT) != 0u;
      if (staged) {                    // the stage is rewritten: the previous tile's bulk stores must have read it
        if (lane == 0) bulk_wait_read_all();
        __syncwarp();
      }
      const bool store = !(elide && (fl & DFLOW_NO_STORE));
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        acc[k] = add_f32x4(b[k], acc[k]);
        if (store) st16(dp + k * 512, acc[k], pol);
        if (staged) sts16(stage + (lane + k * 32) * 16, acc[k]);
      }
      if (staged) fence_proxy_async();
      if ((fl & DFLOW_DEAD_SRC) && !(elide && (fl & DFLOW_SRC_FWD))) {
#pragma unroll
        for (int k = 0; k < 4; ++k) discard_line16(sp + k * 512, v0 + k * 32, vend);
      }
      __syncwarp();   // stage writes before lane 0's bulk stores; a lane's discard before other lanes' later stores to the line
    }
    cur = nxt;
  }
}

// The same for bf16 plans: a unit is 8 elements -- 16 bytes of bf16 in a rank buffer (kind 0) or 32 bytes of fp32
// partials in the shadow (kind 1) -- four units per lane, the running sum as 8 fp32 values per unit in `acc` (the
// kernel's carried registers).  A flow's kinds (source, destination before, destination after) are in its record; the
// sum is rounded to bf16 once, when the flow that completes it stores it to the rank buffer (R12).
template <class PolX>
__device__ __forceinline__ void lean_item_bf16(const ExecParams& P, unsigned int fb, unsigned int fe, unsigned long long off,
                                               unsigned long long tile_unit0, unsigned int lane, char* stage, const PolX& pol,
                                               unsigned long long bulk_pol, uint4 (&acc)[8]) {
  const bool elide = (P.data_fwd & 2u) != 0u, bulk = P.col_bulk != 0u, pf = P.col_pf_dist != 0u;
  const unsigned long long u0 = tile_unit0 + lane, uend = tile_unit0 + 128u;
  // the lane's first unit of rank r's range, in the rank buffer and in the shadow
  auto buf_ptr = [&](unsigned int r) { return rank_ptr(P, r) + off * 2 + u0 * 16; };
  auto sh_ptr = [&](unsigned int r) { return reinterpret_cast<char*>(P.shadow + (unsigned long long)r * P.padded_n + off) + u0 * 32; };
  const uint4* const rec = reinterpret_cast<const uint4*>(P.flows + fb) + 1;
  uint4 cur = __ldg(rec);
  auto first_touches = [&](const uint4& r) {     // raw inputs live in the rank buffers: requested a flow ahead
    if (r.z & DFLOW_SRC_INIT) { const char* q = buf_ptr(r.x & 0xFFFFu); for (int k = 0; k < 4; ++k) prefetch_l1(q + k * 512); }
    if ((r.y & 0xFFu) == 0u && (r.z & DFLOW_DST_INIT)) { const char* q = buf_ptr(r.x >> 16); for (int k = 0; k < 4; ++k) prefetch_l1(q + k * 512); }
  };
  if (pf) first_touches(cur);
  for (unsigned int j = fb; j < fe; ++j) {
    const uint4 nxt = __ldg(rec + 2 * ((j + 1 < fe ? j + 1 : j) - fb));
    const unsigned int src = cur.x & 0xFFFFu, dst = cur.x >> 16, fl = cur.z;
    const unsigned int ksrc = (cur.y >> 8) & 0xFFu, kdin = (cur.y >> 16) & 0xFFu, kdout = cur.y >> 24;
    if (pf && j + 1 < fe) first_touches(nxt);
    if ((cur.y & 0xFFu) != 0u) {       // copy
      if (bulk && (fl & DFLOW_FROM_STAGE)) {
        if (lane == 0) bulk_s2g_hint(rank_ptr(P, dst) + off * 2 + tile_unit0 * 16, stage, 128u * 16u, bulk_pol);
      } else if (ksrc == 0u) {         // bf16 -> bf16: one vector per unit
        const char* sp = buf_ptr(src);
        char* dp = buf_ptr(dst);
#pragma unroll
        for (int k = 0; k < 4; ++k) st16(dp + k * 512, ld16(sp + k * 512, pol.lds, pol.l1), pol);
        __syncwarp();
      } else {                         // fp32 partials -> fp32 partials: two vectors per unit
        const char* sp = sh_ptr(src);
        char* dp = sh_ptr(dst);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint4 x0 = ld16(sp + k * 1024, pol.lds, pol.l1), x1 = ld16(sp + k * 1024 + 16, pol.lds, pol.l1);
          st16(dp + k * 1024, x0, pol);
          st16(dp + k * 1024 + 16, x1, pol);
        }
        __syncwarp();
      }
    } else {                           // reduce
      if (!(fl & DFLOW_SRC_REG)) {     // the source operand: raw bf16 or fp32 partials
        if (ksrc == 0u) {
          const char* sp = buf_ptr(src);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const uint4 r = ld16(sp + k * 512, pol.lds, pol.l1);
            acc[2 * k] = make_uint4(r.x << 16, r.x & 0xFFFF0000u, r.y << 16, r.y & 0xFFFF0000u);
            acc[2 * k + 1] = make_uint4(r.z << 16, r.z & 0xFFFF0000u, r.w << 16, r.w & 0xFFFF0000u);
          }
        } else {
          const char* sp = sh_ptr(src);
#pragma unroll
          for (int k = 0; k < 4; ++k) { acc[2 * k] = ld16(sp + k * 1024, pol.lds, pol.l1); acc[2 * k + 1] = ld16(sp + k * 1024 + 16, pol.lds, pol.l1); }
        }
      }
      const bool staged = bulk && (fl & DFLOW_STAGE_OUT) != 0u && kdout == 0u;
      if (staged) {
        if (lane == 0) bulk_wait_read_all();
        __syncwarp();
      }
      const bool store = !(elide && (fl & DFLOW_NO_STORE));
      const char* dip = kdin ? sh_ptr(dst) : buf_ptr(dst);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        uint4 b0, b1;                  // the destination operand as 8 fp32 bit patterns
        if (kdin) {
          b0 = ld16(dip + k * 1024, pol.ldd, pol.l1);
          b1 = ld16(dip + k * 1024 + 16, pol.ldd, pol.l1);
        } else {
          const uint4 r = ld16(dip + k * 512, pol.ldd, pol.l1);
          b0 = make_uint4(r.x << 16, r.x & 0xFFFF0000u, r.y << 16, r.y & 0xFFFF0000u);
          b1 = make_uint4(r.z << 16, r.z & 0xFFFF0000u, r.w << 16, r.w & 0xFFFF0000u);
        }
        uint4 c0 = add_f32x4(b0, acc[2 * k]), c1 = add_f32x4(b1, acc[2 * k + 1]);
        if (kdout) {
          if (store) { char* dp = sh_ptr(dst); st16(dp + k * 1024, c0, pol); st16(dp + k * 1024 + 16, c1, pol); }
        } else {                       // complete sum: one RNE rounding, to the rank buffer (and the stage)
          uint4 o;
          o.x = f32_to_bf16_rne(__uint_as_float(c0.x)) | (f32_to_bf16_rne(__uint_as_float(c0.y)) << 16);
          o.y = f32_to_bf16_rne(__uint_as_float(c0.z)) | (f32_to_bf16_rne(__uint_as_float(c0.w)) << 16);
          o.z = f32_to_bf16_rne(__uint_as_float(c1.x)) | (f32_to_bf16_rne(__uint_as_float(c1.y)) << 16);
          o.w = f32_to_bf16_rne(__uint_as_float(c1.z)) | (f32_to_bf16_rne(__uint_as_float(c1.w)) << 16);
          if (store) st16(buf_ptr(dst) + k * 512, o, pol);
          if (staged) sts16(stage + (lane + k * 32) * 16, o);
          c0 = make_uint4(o.x << 16, o.x & 0xFFFF0000u, o.y << 16, o.y & 0xFFFF0000u);   // what a load of it would return
          c1 = make_uint4(o.z << 16, o.z & 0xFFFF0000u, o.w << 16, o.w & 0xFFFF0000u);
        }
        acc[2 * k] = c0;
        acc[2 * k + 1] = c1;
      }
      if (staged) fence_proxy_async();
      if ((fl & DFLOW_DEAD_SRC) && !(elide && (fl & DFLOW_SRC_FWD))) {
        if (ksrc == 0u) { const char* sp = buf_ptr(src); for (int k = 0; k < 4; ++k) discard_line16(sp + k * 512, u0 + k * 32, uend); }
        else { const char* sp = sh_ptr(src); for (int k = 0; k < 4; ++k) discard_line32(sp + k * 1024, u0 + k * 32, uend); }
      }
      __syncwarp();
    }
    cur = nxt;
  }
}

template <int MODE, bool MASK_FWD = false>
__global__ void __launch_bounds__(COL_THREADS, CTAS_PER_SM) optcc_wcolumn_kernel(const __grid_constant__ ExecParams P) {
  if (tables_are_stale(P)) return;
  extern __shared__ __align__(128) char s_stage_w[];   // bulk all-gather path: one tile per warp
  const unsigned int lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  char* const stage = s_stage_w + (size_t)warp * P.col_stage_bytes;
  unsigned int overlaps = 0;
  const Pol pol0 = make_policies(P.l2_hints);
  PolL1 pol;                         // a tile is private to its warp for the whole launch: loads and stores through L1
  pol.lds = pol0.lds; pol.ldd = pol0.ldd; pol.st = pol0.st;
  const bool bulk = P.col_bulk != 0;
  bool stage_ok = true;              // contributor masks: every staged set is the full set
  // what the previous flow of the list produced for this lane's vectors (lazy contributor-mask runs: DFLOW_SRC_FWD; data
  // runs: DFLOW_SRC_REG -- a bf16 unit is 8 fp32 values, four units per lane)
  uint4 carry[MODE == MODE_BF16 ? 8 : 4];
  const unsigned long long bulk_pol = make_policy(P.col_bulk_policy);   // L2 policy of the bulk stores
  const bool pf = !is_mask_mode(MODE) && P.col_pf_dist != 0;
  // Items are dealt round-robin to the warps of the grid (neighbouring warps take neighbouring tiles) or, when there
  // are only a few per warp, claimed one at a time through the global ticket (ExecParams.col_chunk, see launch_plan).
  const unsigned long long n_warps = (unsigned long long)gridDim.x * (COL_THREADS / 32);
  const unsigned int CH = P.col_chunk;               // 0: static dealing; else items a warp claims at a time
  // (a warp's first item is always its own number: 4144 claims at the start of the kernel would queue for 0.4 ms)
  unsigned long long it = (unsigned long long)blockIdx.x * (COL_THREADS / 32) + warp, it_end = it + 1;
  for (;; it += CH ? 1 : n_warps) {
    if (CH) {
      if (it == it_end) {
        unsigned long long b = 0;
        if (lane == 0) b = n_warps + atomicAdd(&P.ctrl->ticket, (unsigned long long)CH);
        b = __shfl_sync(0xFFFFFFFFu, b, 0);
        it = b;
        it_end = b + CH;
      }
    }
    if (it >= P.col_n_items) break;
    const uint4 item = __ldg(P.col_items + (it * P.item_stride + P.item_first));
    const unsigned int fb = item.x, fe = item.y;
    const unsigned long long ubeg = (unsigned long long)item.z * P.tile_units, uend = ubeg + item.w;
    DFlow cur = load_record(P.flows + fb);
    if (MASK_FWD && !is_mask_mode(MODE) && item.w == 128u && (ubeg + 128u) * P.unit_elems <= cur.len) {
      // (a full tile inside the region: no ragged end, four vectors / units per lane)
      if (MODE == MODE_F32)
        lean_item_f32(P, fb, fe, cur.off * 4 + ubeg * 16, lane, stage, pol, bulk_pol, ubeg + lane, ubeg + 128u,
                      reinterpret_cast<uint4 (&)[4]>(carry));
      else
        lean_item_bf16(P, fb, fe, cur.off, ubeg, lane, stage, pol, bulk_pol, reinterpret_cast<uint4 (&)[8]>(carry));
      continue;
    }
    if (pf) prefetch_raw<MODE, 32>(P, cur, ubeg, item.w);
    int prev_cls = -1;
    // the tile in bytes of the run's element type (all flows over a region have the region's offset and length)
    bool ragged;
    unsigned long long tile_byte0;
    unsigned int tile_bytes, nv;
    {
      constexpr unsigned long long ESZ = ModeTraits<MODE>::ESIZE, VE = 16 / ESZ;
      const unsigned long long len = cur.len, e0 = ubeg * P.unit_elems;
      unsigned long long e1 = uend * P.unit_elems;
      ragged = e1 > len && (len % VE) != 0;
      if (e1 > len) e1 = len;
      const unsigned long long v0 = e0 / VE, v1 = e1 / VE;     // whole 16-byte vectors of the tile
      tile_byte0 = v0 * 16;
      tile_bytes = (unsigned int)((v1 - v0) * 16);
      const unsigned long long mine0 = v0 + lane;
      nv = mine0 >= v1 ? 0u : (unsigned int)((v1 - mine0 + 31) / 32);
    }
    for (unsigned int j = fb; j < fe; ++j) {
      const DFlow nxt = load_record(P.flows + (j + 1 < fe ? j + 1 : j));
      if (pf && j + 1 < fe) prefetch_raw<MODE, 32>(P, nxt, ubeg, item.w);   // first touches of the next flow
      // fast paths: flows that touch no memory from this lane (see optcc_column_kernel)
      if (MASK_FWD && is_mask_mode(MODE) && !ragged && cur.op == 0 &&
          (cur.flags & (DFLOW_SRC_FWD | DFLOW_DST_INIT | DFLOW_NO_STORE | DFLOW_FINAL | DFLOW_STAGE_OUT)) ==
              (DFLOW_SRC_FWD | DFLOW_DST_INIT | DFLOW_NO_STORE)) {
        constexpr int EB = ModeTraits<MODE>::ESIZE;
        mask_hop_in_registers<EB>(reinterpret_cast<uint4 (&)[4]>(carry), mask_vector(cur.dst < 64 ? 1ull << cur.dst : 0ull, cur.dst >= 64 ? 1ull << (cur.dst - 64) : 0ull, EB),
                                  nv, overlaps);
        cur = nxt;
        continue;
      }
      if (bulk && !ragged && (cur.flags & DFLOW_FROM_STAGE) &&
          !(is_mask_mode(MODE) && P.mask_lazy && (cur.flags & DFLOW_FINAL) && !stage_ok)) {
        if (lane == 0) bulk_s2g_hint(rank_ptr(P, cur.dst) + cur.off * ModeTraits<MODE>::ESIZE + tile_byte0, stage, tile_bytes, bulk_pol);
        cur = nxt;
        continue;
      }
      if (MODE == MODE_BF16) {
        // a copy of fp32 partials moves two vectors per unit, lane i taking vector i instead of unit i: when the
        // lane-to-element mapping changes between consecutive flows the warp synchronises
        const int cls = (cur.op == 1 && cur.ksrc != 0) ? 1 : 0;
        if (prev_cls >= 0 && cls != prev_cls) __syncwarp();
        prev_cls = cls;
      }
      const unsigned int fl = cur.flags;
      if (bulk && (fl & DFLOW_STAGE_OUT)) {
        // the stage is rewritten: the previous tile's bulk stores must have read it
        if (lane == 0) bulk_wait_read_all();
        __syncwarp();
        bool mine = true;
        process_piece<MODE, 32, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, true, stage, false, &mine);
        // this lane's generic-proxy writes (the stage; its earlier stores to ranges the bulk stores will overwrite) are
        // ordered before the async-proxy operations lane 0 issues after the warp barrier
        fence_proxy_async();
        if (is_mask_mode(MODE)) stage_ok = __all_sync(0xFFFFFFFFu, mine) != 0; else __syncwarp();
      } else if (bulk && (fl & DFLOW_FROM_STAGE)) {
        if (is_mask_mode(MODE) && P.mask_lazy && (fl & DFLOW_FINAL) && !stage_ok) {
          process_piece<MODE, 32, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, false, stage, true);
        } else {
          if (lane == 0) {
            constexpr unsigned long long ESZ = ModeTraits<MODE>::ESIZE, VE = 16 / ESZ;
            const unsigned long long e0 = ubeg * P.unit_elems;
            unsigned long long e1 = uend * P.unit_elems;
            if (e1 > cur.len) e1 = cur.len;
            const unsigned long long v0 = e0 / VE, v1 = e1 / VE;
            if (v1 > v0) bulk_s2g_hint(rank_ptr(P, cur.dst) + cur.off * ESZ + v0 * 16, stage, (unsigned int)((v1 - v0) * 16), bulk_pol);
          }
          process_piece<MODE, 32, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, false, nullptr, true);   // (ragged end of a buffer only)
        }
      } else {
        process_piece<MODE, 32, MASK_FWD>(P, cur, ubeg, uend, overlaps, pol, carry, true);
      }
      __syncwarp();   // orders a lane's dead-source discard of a 128-byte line before the other lanes' later stores to it
      cur = nxt;
    }
  }
  if (bulk && lane == 0) bulk_wait_all();   // the stage stays valid until every bulk store has read it
  if (is_mask_mode(MODE)) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) overlaps += __shfl_xor_sync(0xFFFFFFFFu, overlaps, o);
    if (lane == 0 && overlaps) atomicAdd(&P.ctrl->overlap, (unsigned long long)overlaps);
  }
}

// masks[r][e] = {r}: blockIdx.y = rank, 16-byte stores over the rank's padded array; eb = bytes per mask
__global__ void __launch_bounds__(256) optcc_mask_init_kernel(char* masks, unsigned long long padded_n, unsigned int eb) {
  const unsigned int r = blockIdx.y;
  const uint4 v = mask_vector(r < 64 ? 1ull << r : 0ull, r >= 64 ? 1ull << (r - 64) : 0ull, eb);
  uint4* m = reinterpret_cast<uint4*>(masks + (unsigned long long)r * padded_n * eb);
  const unsigned long long nvec = padded_n * eb / 16;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < nvec;
       i += (unsigned long long)gridDim.x * blockDim.x)
    __stcg(m + i, v);
}

// every (rank, element) must hold every rank exactly once: mask == all p bits (PAPER.md:68 (ii))
__global__ void __launch_bounds__(256) optcc_mask_check_kernel(const char* masks, unsigned int p, unsigned long long n,
                                                               unsigned long long padded_n, unsigned int eb, Ctrl* ctrl) {
  const unsigned int r = blockIdx.y;
  const unsigned long long full0 = p >= 64 ? ~0ull : ((1ull << p) - 1ull);
  const unsigned long long full1 = p > 64 ? (p >= 128 ? ~0ull : ((1ull << (p - 64)) - 1ull)) : 0ull;
  const uint4 F = mask_vector(full0, full1, eb);
  const uint4* m = reinterpret_cast<const uint4*>(masks + (unsigned long long)r * padded_n * eb);
  const unsigned int epv = 16 / eb;                                  // elements per vector
  const unsigned long long nvec = (n + epv - 1) / epv;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned long long bad = 0, first = ~0ull;
  for (unsigned long long i0 = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i0 < nvec; i0 += 4 * stride) {
    uint4 vv[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) vv[q] = i0 + q * stride < nvec ? __ldcg(m + i0 + q * stride) : F;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const unsigned long long i = i0 + q * stride;
      if (i >= nvec) break;
      const unsigned int dx = vv[q].x ^ F.x, dy = vv[q].y ^ F.y, dz = vv[q].z ^ F.z, dw = vv[q].w ^ F.w;
      if ((dx | dy | dz | dw) == 0u) continue;
      const unsigned int d[4] = {dx, dy, dz, dw};
      for (unsigned int j = 0; j < epv; ++j) {                      // rare path: locate the wrong elements
        const unsigned long long e = i * epv + j;
        if (e >= n) break;
        bool wrong;
        if (eb == 2) wrong = ((d[j >> 1] >> ((j & 1u) * 16)) & 0xFFFFu) != 0u;
        else if (eb == 4) wrong = d[j] != 0u;
        else if (eb == 8) wrong = (d[2 * j] | d[2 * j + 1]) != 0u;
        else wrong = true;
        if (wrong) { ++bad; const unsigned long long g = (unsigned long long)r * n + e; first = first < g ? first : g; }
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bad += __shfl_xor_sync(0xFFFFFFFFu, bad, o);
    unsigned long long other = __shfl_xor_sync(0xFFFFFFFFu, first, o);
    first = first < other ? first : other;
  }
  if ((threadIdx.x & 31) == 0 && bad) {
    atomicAdd(&ctrl->bad, bad);
    atomicMin(&ctrl->first_bad, first);
  }
}

}  // namespace

// =====================================================================================================
// Host side
// =====================================================================================================

namespace {
// Which plan's tables a workspace currently holds (by workspace address).  Contents are the caller's to keep intact
// between calls; after reusing the memory for something else, call optcc_prepare again.
std::mutex g_ws_mutex;
std::unordered_map<void*, uint64_t> g_ws_owner;
std::atomic<uint64_t> g_next_id{1};
}  // namespace

namespace {
// Page-locked host memory for the one big table that is built and uploaded again for every plan (the column executor's
// records: 31 MB at C4 / k = 32).  A cudaMemcpyAsync from pageable memory is staged through the driver's bounce buffers
// ON THE CALLING THREAD; from page-locked memory it is one DMA the host does not wait for.  Blocks go back to a small
// process-wide cache (cudaHostAlloc costs more than the copy it saves; a job that plans every step reuses the block).
// Without a driver (planning on a CPU box: optcc_column_tables), or when the calling thread forbids allocating CUDA
// calls (optcc_execute_static), the memory is pageable, from optcc_raw_alloc.
struct PinnedBlock { void* p; size_t bytes; };
std::mutex g_pinned_mutex;
std::vector<PinnedBlock> g_pinned_cache;
constexpr size_t PINNED_MIN = size_t(1) << 20, PINNED_CACHE_BLOCKS = 4, PINNED_CACHE_MAX = size_t(512) << 20;
thread_local bool tl_no_cuda_alloc = false;

void* pinned_alloc(size_t bytes) {                       // nullptr: use pageable memory
  if (bytes < PINNED_MIN || tl_no_cuda_alloc) return nullptr;
  {
    std::lock_guard<std::mutex> lock(g_pinned_mutex);
    size_t best = SIZE_MAX;
    for (size_t i = 0; i < g_pinned_cache.size(); ++i)
      if (g_pinned_cache[i].bytes >= bytes && g_pinned_cache[i].bytes <= 2 * bytes &&
          (best == SIZE_MAX || g_pinned_cache[i].bytes < g_pinned_cache[best].bytes)) best = i;
    if (best != SIZE_MAX) {
      void* q = g_pinned_cache[best].p;
      g_pinned_cache.erase(g_pinned_cache.begin() + best);
      return q;
    }
  }
  // Page-locking costs far more than the copy it speeds up (measured: 40 ms for 31 MB against 3 ms saved), so it only
  // pays for a process that builds big tables again and again and gets its block back from the cache: the first big
  // table of a process stays pageable.
  static std::atomic<unsigned> big_tables{0};
  if (big_tables.fetch_add(1, std::memory_order_relaxed) == 0) return nullptr;
  void* q = nullptr;
  if (cudaHostAlloc(&q, bytes, cudaHostAllocDefault) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return q;
}

void pinned_free(void* q, size_t bytes) {
  {
    std::lock_guard<std::mutex> lock(g_pinned_mutex);
    // the newest block stays, the oldest ones go (a job that moves on to another plan shape must find ITS blocks cached;
    // cudaFreeHost waits for the device, so it must not happen on every step)
    if (bytes <= PINNED_CACHE_MAX) {
      g_pinned_cache.push_back(PinnedBlock{q, bytes});
      size_t total = 0;
      for (const auto& b : g_pinned_cache) total += b.bytes;
      while (g_pinned_cache.size() > PINNED_CACHE_BLOCKS || total > PINNED_CACHE_MAX) {
        total -= g_pinned_cache.front().bytes;
        cudaFreeHost(g_pinned_cache.front().p);
        g_pinned_cache.erase(g_pinned_cache.begin());
      }
      return;
    }
  }
  cudaFreeHost(q);
}

template <class T>
class HostTable {
 public:
  HostTable() = default;
  HostTable(const HostTable&) = delete;
  HostTable& operator=(const HostTable&) = delete;
  ~HostTable() { release(); }
  void release() {
    if (p_) { if (pinned_) pinned_free(p_, cap_ * sizeof(T)); else optcc_raw_free(p_, cap_ * sizeof(T)); }
    p_ = nullptr; n_ = cap_ = 0; pinned_ = false;
  }
  void resize_uninit(size_t n) {          // contents undefined; throws std::bad_alloc
    if (n > cap_) {
      release();
      void* q = pinned_alloc(n * sizeof(T));
      pinned_ = q != nullptr;
      if (!q) q = optcc_raw_alloc(n * sizeof(T));
      if (!q) throw std::bad_alloc();
      p_ = static_cast<T*>(q);
      cap_ = n;
    }
    n_ = n;
  }
  bool pinned() const { return pinned_; }
  size_t size() const { return n_; }
  bool empty() const { return n_ == 0; }
  T* data() { return p_; }
  const T* data() const { return p_; }
  T& operator[](size_t i) { return p_[i]; }
  const T& operator[](size_t i) const { return p_[i]; }
 private:
  T* p_ = nullptr;
  size_t n_ = 0, cap_ = 0;
  bool pinned_ = false;
};
}  // namespace

struct optcc_exec_state {
  int device = -1;
  int sm_count = 0;
  int coop = 0;
  uint32_t G = 0;                 // executor grid (CTAs)
  uint64_t id = 0;                // process-unique id of this plan's device tables (see g_ws_owner)
  unsigned long long stamp_host = 0;   // table_stamp(id), the value upload_tables writes into the control block
  std::vector<DFlow> dflows;
  std::vector<Slice> slices;      // [n_steps][G + 1]
  // dataflow executor
  uint32_t G_df = 0;              // grid of the dataflow kernel
  bool df_ok = false;             // counters fit 32-bit indices
  bool big_ops = false;           // average tile-op >= 1792 units (decides the ring depth)
  bool lazy_masks = false;        // the verifier needs no init / check passes (see assign_mask_flags)
  bool built = false;             // every table of this state is complete (set last; cleared on any failure)
  bool host_built = false;        // the device-independent tables are complete
  std::vector<DDep> deps;         // [n_flows]
  std::vector<TileOp> ops;        // [n_tile_ops], table order
  std::vector<uint64_t> step_op_begin;   // [n_steps + 1]
  // column executor
  bool column = false;
  HostTable<DFlow> col_dflows;           // the executed flows, region by region (chain order inside a region)
  cudaEvent_t uploaded = nullptr;        // recorded after an upload from page-locked tables: they may not be recycled before it
  std::vector<uint32_t> col_reg_begin;   // [regions + 1]
  std::vector<uint4> col_items;          // (first flow, end flow, tile, units in the tile)
  std::vector<uint4> col_items_mask;     // the verifier's items when its tile size differs (plan's mask_tile_units)
};

// The stamp a workspace carries while it holds the tables of state `id`: kernels compare it with their launch parameter.
static inline unsigned long long table_stamp(uint64_t id) { return 0x4F50544343000000ull ^ (id * 0x9E3779B97F4A7C15ull); }

void optcc_exec_state_free(optcc_exec_state* s) {
  if (s) {   // the workspaces that held this plan's tables no longer count as prepared
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    for (auto it = g_ws_owner.begin(); it != g_ws_owner.end();)
      it = it->second == s->id ? g_ws_owner.erase(it) : std::next(it);
  }
  if (s && s->uploaded) {   // a copy from the page-locked table may still be in flight: its block goes back to a cache
    cudaEventSynchronize(s->uploaded);
    cudaEventDestroy(s->uploaded);
    cudaGetLastError();
  }
  delete s;
}

namespace {

template <int MODE>
int df_kernel_occupancy(int* out) {
  const size_t dyn = size_t(BULK_SMEM_PER_AGENT) * DF_SLOTS;   // sized for the bulk-copy path
  CU_TRY(cudaFuncSetAttribute(optcc_dataflow_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, optcc_dataflow_kernel<MODE>, DF_THREADS, dyn));
  return OPTCC_OK;
}

// Dataflow tables: tile-ops in table order and, per flow, the completion counts its ranges must have reached.
// Per (rank, region) the accesses are ordered as in the table; a read waits for the last write before it, a write
// for every earlier access (see optcc_dataflow_kernel).
void build_dataflow_tables(optcc_plan_t* pl, optcc_exec_state* st) {
  const optcc_plan_info_t& in = pl->info;
  const uint64_t A = in.unit_elems, TU = pl->tile_units, nr = pl->region_offs.size();
  st->df_ok = uint64_t(in.p) * pl->tiles_per_rank < (uint64_t(1) << 32) && pl->n_tile_ops < (uint64_t(1) << 40);
  {
    uint64_t units = 0;
    for (const auto& f : pl->flows) units += (f.len + A - 1) / A;
    st->big_ops = pl->n_tile_ops && units / pl->n_tile_ops >= 1792;
  }
  if (!st->df_ok) return;
  struct RangeState { uint32_t count, lastw, readers; };   // accesses so far, position after the last write, reads since it
  std::vector<RangeState> rs(size_t(in.p) * nr, RangeState{0, 0, 0});
  std::vector<uint8_t> sole_reader(in.n_flows, 0);       // the flow is the first reader of its source since the last write
  st->deps.resize(in.n_flows);
  st->ops.resize(pl->n_tile_ops);
  TileOp* op_out = st->ops.data();
  st->step_op_begin.assign(in.n_steps + 1, 0);
  uint32_t step = 0;
  for (uint32_t i = 0; i < in.n_flows; ++i) {
    const optcc_flow_t& f = pl->flows[i];
    while (step < f.step) st->step_op_begin[++step] = uint64_t(op_out - st->ops.data());
    const size_t reg = pl->flow_region[i];
    const size_t ls = size_t(f.src) * nr + reg, ld = size_t(f.dst) * nr + reg;
    DDep d;
    d.csrc = uint32_t(uint64_t(f.src) * pl->tiles_per_rank + pl->region_tile0[reg]);
    d.cdst = uint32_t(uint64_t(f.dst) * pl->tiles_per_rank + pl->region_tile0[reg]);
    RangeState& S = rs[ls];
    d.need_src = S.lastw;
    S.count++;
    sole_reader[i] = S.readers++ == 0;
    RangeState& D = rs[ld];
    d.need_dst = D.count;
    D.lastw = ++D.count;
    D.readers = 0;
    st->deps[i] = d;
    const uint64_t ntiles = ((f.len + A - 1) / A + TU - 1) / TU;
    for (uint64_t t = 0; t < ntiles; ++t) *op_out++ = TileOp{i, uint32_t(t)};
  }
  while (step < in.n_steps) st->step_op_begin[++step] = uint64_t(op_out - st->ops.data());
  // dead sources: walking the table backwards, the source range of flow i is dead after i has read it iff the next
  // access to that (rank, region) is a plain overwrite by a copy flow (a reduce would still read it, a read needs
  // it, and no further access means it is a final result).  Only reduce flows act on the flag (their sources are the
  // partial sums and raw inputs that the all-gather overwrites later).
  enum : uint8_t { NEXT_NONE = 0, NEXT_READ, NEXT_COPY_WRITE, NEXT_REDUCE_WRITE };
  std::vector<uint8_t> next(size_t(in.p) * nr, NEXT_NONE);
  for (uint32_t i = in.n_flows; i-- > 0;) {
    const optcc_flow_t& f = pl->flows[i];
    const size_t reg = pl->flow_region[i];
    const size_t ls = size_t(f.src) * nr + reg, ld = size_t(f.dst) * nr + reg;
    // (first and last reader since the last write = the only one: no other flow may still be reading the range)
    // (not for truncated schedules, step_limit: the overwrite that makes the range dead might never run)
    st->dflows[i].flags = (!pl->opts.no_discard && !pl->opts.step_limit && f.op == OPTCC_OP_REDUCE && next[ls] == NEXT_COPY_WRITE && sole_reader[i]) ? 1u : 0u;
    next[ld] = f.op == OPTCC_OP_COPY ? NEXT_COPY_WRITE : NEXT_REDUCE_WRITE;
    next[ls] = NEXT_READ;
  }
}

// Lazy verifier (range_mask_lazy; the planner decides, info.lazy_verify): the executed part of the table writes every
// (rank, region) at least once, so no mask the run reads or leaves behind is one it has not written -- the arrays
// need no initialising pass and the last writer of every range checks the final mask.  Sets the DFLOW_*_INIT / FINAL
// bits; otherwise the flags stay clear and optcc_verify initialises and checks the arrays with separate passes.
void assign_mask_flags(optcc_plan_t* pl, optcc_exec_state* st) {
  const optcc_plan_info_t& in = pl->info;
  st->lazy_masks = false;
  if (!in.lazy_verify) return;
  const uint32_t steps = pl->opts.step_limit ? std::min(pl->opts.step_limit, in.n_steps) : in.n_steps;
  const uint32_t nf = pl->step_begin[steps];            // flows of the executed steps
  const size_t nr = pl->region_offs.size();
  std::vector<uint8_t> written(size_t(in.p) * nr, 0);
  const optcc_rawvec<uint32_t>& reg = pl->flow_region;
  for (uint32_t i = 0; i < nf; ++i) {                   // forwards: has the range been written before flow i?
    const optcc_flow_t& f = pl->flows[i];
    uint32_t fl = 0;
    if (!written[size_t(f.src) * nr + reg[i]]) fl |= DFLOW_SRC_INIT;
    if (!written[size_t(f.dst) * nr + reg[i]]) fl |= DFLOW_DST_INIT;
    written[size_t(f.dst) * nr + reg[i]] = 1;
    st->dflows[i].flags |= fl;
  }
  std::fill(written.begin(), written.end(), 0);
  for (uint32_t i = nf; i-- > 0;) {                     // backwards: is the range written after flow i?
    const optcc_flow_t& f = pl->flows[i];
    if (!written[size_t(f.dst) * nr + reg[i]]) st->dflows[i].flags |= DFLOW_FINAL;
    written[size_t(f.dst) * nr + reg[i]] = 1;
  }
  st->lazy_masks = true;
}

// =====================================================================================================
// Column executor tables.  The flows of the executed steps are stored region by region (a stable parallel counting
// sort of the table by region: table order is kept inside a region); then every region's list is finished on its own
// -- lists are independent, so this runs on a few host threads:
//   * order: any order that respects the data dependencies inside the column gives the same bits; the
//     list is rearranged chain by chain (a flow is followed by the flow that reads what it wrote whenever that one is
//     ready), so that a CTA keeps one partial tile live instead of one per interleaved chain (C4: the collect /
//     distribute flows of 16 servers interleave in table order);
//   * storage kinds of bf16 plans (fp32 shadow while 1 < contributors < p);
//   * DFLOW_SRC_INIT / DST_INIT (first touches), DFLOW_FINAL (last writes), DFLOW_DEAD_SRC, and the bulk all-gather
//     flags DFLOW_STAGE_OUT / FROM_STAGE;
//   * coverage: the lazy verifier needs every rank's range written by the list.
// Regions of one class (same part and section, another segment) have the same list up to the offset: the work is done
// once per class and copied after an element-wise check of (src, dst, op).
// =====================================================================================================
struct ColScratch {
  std::vector<uint16_t> cnt;
  std::vector<uint8_t> written, next, bulkw, sole, done;
  std::vector<uint32_t> readers, val, consumers;
  std::vector<int32_t> last_writer, rd_head, rd_next;
  std::vector<uint32_t> e_from, e_to, succ_begin, succ, indeg, order, heap;
  std::vector<DFlow> tmp, rep_final;
  std::vector<uint64_t> rep_key;     // src, dst, op of the representative's flows, table order
  std::vector<uint32_t> rep_order;
  bool rep_valid = false, rep_covered = false;
  void init(uint32_t p) {
    cnt.resize(p); written.resize(p); next.resize(p); bulkw.resize(p); readers.resize(p); val.resize(p);
    last_writer.resize(p); rd_head.resize(p);
  }
};

inline uint64_t flow_key(const DFlow& f) { return (uint64_t)f.src << 32 | (uint64_t)f.dst << 8 | f.op; }

// chain-by-chain order of one list (see above); out: sc.order[0..n)
void chain_order(const DFlow* L, uint32_t n, uint32_t p, ColScratch& sc) {
  sc.e_from.clear(); sc.e_to.clear();
  sc.rd_next.assign(n, -1);
  std::fill(sc.last_writer.begin(), sc.last_writer.end(), -1);
  std::fill(sc.rd_head.begin(), sc.rd_head.end(), -1);
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t s = L[i].src, d = L[i].dst;
    const int32_t lws = sc.last_writer[s], lwd = sc.last_writer[d];
    if (lws >= 0) { sc.e_from.push_back(lws); sc.e_to.push_back(i); }                  // read after write
    if (lwd >= 0 && lwd != lws) { sc.e_from.push_back(lwd); sc.e_to.push_back(i); }    // write after write (a reduce also reads)
    for (int32_t r = sc.rd_head[d]; r >= 0; r = sc.rd_next[r]) { sc.e_from.push_back(r); sc.e_to.push_back(i); }   // write after read
    sc.rd_head[d] = -1;
    sc.rd_next[i] = sc.rd_head[s];
    sc.rd_head[s] = (int32_t)i;
    sc.last_writer[d] = (int32_t)i;
  }
  const size_t ne = sc.e_from.size();
  sc.succ_begin.assign(size_t(n) + 1, 0);
  sc.indeg.assign(n, 0);
  for (size_t e = 0; e < ne; ++e) { sc.succ_begin[sc.e_from[e] + 1]++; sc.indeg[sc.e_to[e]]++; }
  for (uint32_t i = 0; i < n; ++i) sc.succ_begin[i + 1] += sc.succ_begin[i];
  sc.succ.resize(ne);
  {
    std::vector<uint32_t>& pos = sc.heap;      // (borrowed as a cursor array)
    pos.assign(sc.succ_begin.begin(), sc.succ_begin.end() - 1);
    for (size_t e = 0; e < ne; ++e) sc.succ[pos[sc.e_from[e]]++] = sc.e_to[e];
  }
  sc.done.assign(n, 0);
  sc.order.resize(n);
  std::vector<uint32_t>& heap = sc.heap;       // min-heap of ready flows (lazy deletion through done[])
  heap.clear();
  auto cmp = [](uint32_t a, uint32_t b) { return a > b; };
  for (uint32_t i = 0; i < n; ++i) if (sc.indeg[i] == 0) heap.push_back(i);
  std::make_heap(heap.begin(), heap.end(), cmp);
  int64_t last = -1;
  for (uint32_t k = 0; k < n; ++k) {
    int64_t pick = -1;
    if (last >= 0) {   // prefer the flow that reads what `last` wrote, then another flow into the same destination
      const uint32_t d = L[last].dst;
      int64_t same_dst = -1;
      for (uint32_t e = sc.succ_begin[last]; e < sc.succ_begin[last + 1]; ++e) {
        const uint32_t v = sc.succ[e];
        if (sc.done[v] || sc.indeg[v] != 0) continue;
        if (L[v].src == d) { if (pick < 0 || v < pick) pick = v; }
        else if (L[v].dst == d) { if (same_dst < 0 || v < same_dst) same_dst = v; }
      }
      if (pick < 0) pick = same_dst;
    }
    if (pick < 0) {
      while (sc.done[heap.front()]) { std::pop_heap(heap.begin(), heap.end(), cmp); heap.pop_back(); }
      pick = heap.front();
      std::pop_heap(heap.begin(), heap.end(), cmp);
      heap.pop_back();
    }
    sc.order[k] = (uint32_t)pick;
    sc.done[pick] = 1;
    for (uint32_t e = sc.succ_begin[pick]; e < sc.succ_begin[pick + 1]; ++e) {
      const uint32_t v = sc.succ[e];
      if (--sc.indeg[v] == 0) { heap.push_back(v); std::push_heap(heap.begin(), heap.end(), cmp); }
    }
    last = pick;
  }
}

struct ColBuildOpts { uint32_t p; bool bf16, discard, bulk, reorder; };

// Finish one list in place (L holds the region's flows in table order, flags and kinds clear).  Returns whether every
// rank's range is written by the list.
bool finish_region(DFlow* L, uint32_t n, const ColBuildOpts& o, ColScratch& sc) {
  const uint32_t p = o.p;
  // the same list as the class representative?  then its order, kinds and flags apply
  bool same = sc.rep_valid && sc.rep_key.size() == n;
  for (uint32_t i = 0; i < n && same; ++i) same = sc.rep_key[i] == flow_key(L[i]);
  if (same) {
    sc.tmp.assign(L, L + n);
    for (uint32_t j = 0; j < n; ++j) {
      DFlow f = sc.tmp[sc.rep_order[j]];
      const DFlow& r = sc.rep_final[j];
      f.ksrc = r.ksrc; f.kdin = r.kdin; f.kdout = r.kdout; f.flags = r.flags;
      L[j] = f;
    }
    return sc.rep_covered;
  }
  sc.rep_key.resize(n);
  for (uint32_t i = 0; i < n; ++i) sc.rep_key[i] = flow_key(L[i]);
  if (o.reorder && n > 2) {
    chain_order(L, n, p, sc);
    sc.tmp.assign(L, L + n);
    for (uint32_t j = 0; j < n; ++j) L[j] = sc.tmp[sc.order[j]];
    sc.rep_order = sc.order;
  } else {
    sc.rep_order.resize(n);
    for (uint32_t j = 0; j < n; ++j) sc.rep_order[j] = j;
  }
  // forwards: first touches, storage kinds, sole readers
  std::fill(sc.written.begin(), sc.written.end(), 0);
  std::fill(sc.readers.begin(), sc.readers.end(), 0);
  std::fill(sc.cnt.begin(), sc.cnt.end(), 1);
  sc.sole.resize(n);
  auto kind_of = [&](uint32_t c) -> unsigned char { return (c == 1 || c >= p) ? OPTCC_KIND_BUF : OPTCC_KIND_F32; };
  uint32_t covered = 0;
  for (uint32_t i = 0; i < n; ++i) {
    DFlow& f = L[i];
    unsigned int fl = 0;
    if (!sc.written[f.src]) fl |= DFLOW_SRC_INIT;
    if (!sc.written[f.dst]) fl |= DFLOW_DST_INIT;
    sc.sole[i] = sc.readers[f.src]++ == 0;
    sc.readers[f.dst] = 0;
    covered += !sc.written[f.dst];
    sc.written[f.dst] = 1;
    const uint32_t cs = sc.cnt[f.src], cd = sc.cnt[f.dst], out = f.op == OPTCC_OP_REDUCE ? cs + cd : cs;
    if (o.bf16) { f.ksrc = kind_of(cs); f.kdin = kind_of(cd); f.kdout = kind_of(out); }
    sc.cnt[f.dst] = (uint16_t)std::min<uint32_t>(out, 65535);
    f.flags = fl;
  }
  // backwards: last writes; dead sources (the flow is the only reader of its source range since the last write and
  // the next access to that range is a plain overwrite by a copy flow: only reduce flows act on it)
  enum : uint8_t { NEXT_NONE = 0, NEXT_READ, NEXT_COPY_WRITE, NEXT_REDUCE_WRITE };
  std::fill(sc.next.begin(), sc.next.end(), (uint8_t)NEXT_NONE);
  std::fill(sc.written.begin(), sc.written.end(), 0);
  for (uint32_t i = n; i-- > 0;) {
    DFlow& f = L[i];
    if (!sc.written[f.dst]) f.flags |= DFLOW_FINAL;
    sc.written[f.dst] = 1;
    const bool dead = f.op == OPTCC_OP_REDUCE && sc.next[f.src] == NEXT_COPY_WRITE && sc.sole[i];
    if (o.discard && dead) f.flags |= DFLOW_DEAD_SRC;
    // the verifier's forwarding (lazy contributor-mask runs only): the dead source was written by the flow just before
    // this one, so the sets are still in the thread's registers -- and that flow need not store them, unless its
    // result is a final value or the staged tile
    if (dead && i > 0 && L[i - 1].dst == f.src) {
      f.flags |= DFLOW_SRC_FWD;
    }
    // data runs: the source range holds what the reduce flow just before this one stored -- with the same threads on the
    // same vectors (one-round tiles, ExecParams.data_fwd) the operand is still in registers
    if (f.op == OPTCC_OP_REDUCE && i > 0 && L[i - 1].op == OPTCC_OP_REDUCE && L[i - 1].dst == f.src) f.flags |= DFLOW_SRC_REG;
    sc.next[f.dst] = f.op == OPTCC_OP_COPY ? NEXT_COPY_WRITE : NEXT_REDUCE_WRITE;
    sc.next[f.src] = NEXT_READ;
  }

  // Bulk all-gather path (data runs): find the reduce flows whose sum later copy flows distribute (DFLOW_STAGE_OUT: the
  // CTA keeps the tile in shared memory) and the copy flows whose source range holds exactly the staged tile at that
  // point (DFLOW_FROM_STAGE: one cp.async.bulk store).  Value numbering: a reduce gives its destination a new value,
  // a copy gives it the source's value.  One stage: a new sum is only staged when every copy of the previous one has
  // been issued.  A list in which a range written by a bulk store is touched again by any later flow (never the case
  // in an AllReduce plan: the all-gather's copies are final) keeps the LDG / STG path entirely.
  if (o.bulk) {
    for (uint32_t i = 0; i < p; ++i) sc.val[i] = i;
    sc.consumers.assign(size_t(p) + n, 0);
    uint32_t next_id = p;
    for (uint32_t i = 0; i < n; ++i) {
      const DFlow& f = L[i];
      if (f.op == OPTCC_OP_REDUCE) sc.val[f.dst] = next_id++;
      else { sc.consumers[sc.val[f.src]]++; sc.val[f.dst] = sc.val[f.src]; }
    }
    for (uint32_t i = 0; i < p; ++i) sc.val[i] = i;
    std::fill(sc.bulkw.begin(), sc.bulkw.end(), 0);
    next_id = p;
    uint32_t staged = UINT32_MAX, pending = 0;
    bool ok = true;
    for (uint32_t i = 0; i < n && ok; ++i) {
      DFlow& f = L[i];
      if (f.op == OPTCC_OP_REDUCE) {
        if (sc.bulkw[f.src] || sc.bulkw[f.dst]) { ok = false; break; }
        const uint32_t id = next_id++;
        sc.val[f.dst] = id;
        if (sc.consumers[id] && pending == 0 && (!o.bf16 || f.kdout == OPTCC_KIND_BUF)) {
          f.flags |= DFLOW_STAGE_OUT;
          staged = id;
          pending = sc.consumers[id];
        }
      } else {
        if (sc.val[f.src] == staged && (!o.bf16 || (f.ksrc == OPTCC_KIND_BUF && f.kdout == OPTCC_KIND_BUF))) {
          if (sc.bulkw[f.dst]) { ok = false; break; }
          f.flags |= DFLOW_FROM_STAGE;
          sc.bulkw[f.dst] = 1;
          --pending;
        } else if (sc.bulkw[f.src] || sc.bulkw[f.dst]) {
          ok = false;
          break;
        } else if (sc.val[f.src] == staged) {
          --pending;
        }
        sc.val[f.dst] = sc.val[f.src];
      }
    }
    if (!ok) for (uint32_t i = 0; i < n; ++i) L[i].flags &= ~(DFLOW_STAGE_OUT | DFLOW_FROM_STAGE);
  }
  for (uint32_t i = 1; i < n; ++i) {
    if (!(L[i].flags & DFLOW_SRC_FWD)) continue;
    if (L[i - 1].flags & DFLOW_FROM_STAGE) L[i].flags &= ~DFLOW_SRC_FWD;      // (stored by cp.async.bulk: not in registers)
    else if (!(L[i - 1].flags & (DFLOW_FINAL | DFLOW_STAGE_OUT))) L[i - 1].flags |= DFLOW_NO_STORE;
  }
  sc.rep_final.assign(L, L + n);
  sc.rep_covered = covered == p;
  sc.rep_valid = true;
  return sc.rep_covered;
}

// Finish a list from scratch (no representative to compare with).
inline bool finish_fresh(DFlow* L, uint32_t n, const ColBuildOpts& o, ColScratch& sc) {
  sc.rep_valid = false;
  return finish_region(L, n, o, sc);
}

// Builds col_dflows / col_reg_begin / col_items; sets *all_covered (every rank's range of every region is written by
// the executed steps -- what the lazy verifier needs).
void build_column_state(optcc_plan_t* pl, optcc_exec_state* st, bool* all_covered) {
  const optcc_plan_info_t& in = pl->info;
  const uint64_t A = in.unit_elems, TU = pl->tile_units;
  const size_t nr = pl->region_offs.size();
  const uint32_t steps = pl->opts.step_limit ? std::min(pl->opts.step_limit, in.n_steps) : in.n_steps;
  const uint32_t nf = pl->step_begin[steps];
  ColBuildOpts o;
  o.p = in.p;
  o.bf16 = in.dtype == OPTCC_BF16;
  o.discard = !pl->opts.no_discard && !pl->opts.step_limit;   // (a truncated schedule: the overwrite that makes a range dead might never run)
  o.bulk = pl->opts.copy_path != 1;
  o.reorder = pl->opts.col_order != 1;
  // classes: regions of the same part and section (another segment)
  std::vector<uint32_t> cls_begin, cls_regions;
  {
    uint32_t ncls = 0;
    for (uint32_t c : pl->region_class) ncls = std::max(ncls, c + 1);
    cls_begin.assign(size_t(ncls) + 1, 0);
    for (uint32_t c : pl->region_class) cls_begin[c + 1]++;
    for (uint32_t c = 0; c < ncls; ++c) cls_begin[c + 1] += cls_begin[c];
    cls_regions.resize(nr);
    std::vector<uint32_t> pos(cls_begin.begin(), cls_begin.end() - 1);
    for (size_t r = 0; r < nr; ++r) cls_regions[pos[pl->region_class[r]]++] = (uint32_t)r;
  }
  const size_t ncls = cls_begin.size() - 1;
  std::atomic<uint32_t> uncovered{0};
  // Complete schedules: every rule of PLAN_SPEC 4 places the flows of segment b at steps b P + (something that does not
  // depend on b), so the regions of one class have the SAME list up to offset and length.  Only the list of each
  // class's first region is gathered from the table and finished; the others are copies with their own range.
  bool fast = steps == in.n_steps;
  for (size_t c = 0; c < ncls && fast; ++c)
    for (uint32_t q = cls_begin[c]; q < cls_begin[c + 1]; ++q)
      if (pl->region_flows[cls_regions[q]] != pl->region_flows[cls_regions[cls_begin[c]]]) { fast = false; break; }
  if (fast) {
    st->col_reg_begin.assign(nr + 1, 0);
    for (size_t r = 0; r < nr; ++r) st->col_reg_begin[r + 1] = st->col_reg_begin[r] + pl->region_flows[r];
    st->col_dflows.resize_uninit(nf);
    // gather the lists (table order) of every class's first region -- and of its last one, which is compared with the
    // first before anything is replicated -- straight into their place in col_dflows
    std::vector<uint32_t> fill(nr, UINT32_MAX);            // next free position of a gathered list
    for (size_t c = 0; c < ncls; ++c)
      if (cls_begin[c] < cls_begin[c + 1]) {
        const uint32_t r0 = cls_regions[cls_begin[c]], r1 = cls_regions[cls_begin[c + 1] - 1];
        fill[r0] = st->col_reg_begin[r0];
        fill[r1] = st->col_reg_begin[r1];
      }
    const uint32_t* reg = pl->flow_region.data();
    for (uint32_t i = 0; i < nf; ++i) {
      uint32_t& pos = fill[reg[i]];
      if (pos == UINT32_MAX) continue;
      const optcc_flow_t& f = pl->flows[i];
      DFlow d;
      d.off = f.off; d.len = f.len; d.src = f.src; d.dst = f.dst; d.op = f.op;
      d.ksrc = d.kdin = d.kdout = 0; d.flags = 0; d.pad1 = 0;
      st->col_dflows[pos++] = d;
    }
    for (size_t c = 0; c < ncls && fast; ++c) {
      if (cls_begin[c] == cls_begin[c + 1]) continue;
      const uint32_t r0 = cls_regions[cls_begin[c]], r1 = cls_regions[cls_begin[c + 1] - 1];
      const DFlow* a = st->col_dflows.data() + st->col_reg_begin[r0];
      const DFlow* b = st->col_dflows.data() + st->col_reg_begin[r1];
      for (uint32_t j = 0; j < pl->region_flows[r0] && fast; ++j) fast = flow_key(a[j]) == flow_key(b[j]);
    }
  }
  if (fast) {
    optcc_parallel_chunks(ncls, nf, [&](size_t c) {
      if (cls_begin[c] == cls_begin[c + 1]) return;
      ColScratch sc;
      sc.init(in.p);
      const uint32_t r0 = cls_regions[cls_begin[c]];
      const uint32_t n = pl->region_flows[r0];
      if (n == 0) { uncovered.fetch_add(cls_begin[c + 1] - cls_begin[c], std::memory_order_relaxed); return; }
      DFlow* L0 = st->col_dflows.data() + st->col_reg_begin[r0];
      const bool cov = finish_fresh(L0, n, o, sc);
      if (!cov) uncovered.fetch_add(cls_begin[c + 1] - cls_begin[c], std::memory_order_relaxed);
      for (uint32_t q = cls_begin[c] + 1; q < cls_begin[c + 1]; ++q) {
        const uint32_t r = cls_regions[q];
        DFlow* L = st->col_dflows.data() + st->col_reg_begin[r];
        const uint64_t off = pl->region_offs[r], len = pl->region_len[r];
        for (uint32_t j = 0; j < n; ++j) {
          DFlow f = L0[j];
          f.off = off;
          f.len = len;
          L[j] = f;
        }
      }
    });
  } else {
    // ---- general path (truncated schedules): parallel stable counting sort of the table by region, then every list
    // finished on its own, reusing the class's first list where it is the same ----
    const size_t n_chunks = std::max<size_t>(1, std::min<size_t>(32, nf / 4096));
    auto chunk_lo = [&](size_t c) { return uint32_t(uint64_t(nf) * c / n_chunks); };
    std::vector<uint32_t> hist(n_chunks * nr, 0);
    optcc_parallel_chunks(n_chunks, nf, [&](size_t c) {
      uint32_t* h = hist.data() + c * nr;
      const uint32_t* reg = pl->flow_region.data();
      for (uint32_t i = chunk_lo(c); i < chunk_lo(c + 1); ++i) h[reg[i]]++;
    });
    st->col_reg_begin.assign(nr + 1, 0);
    for (size_t r = 0; r < nr; ++r) {          // hist[c][r] becomes the first position of chunk c's flows of region r
      uint32_t pos = st->col_reg_begin[r];
      for (size_t c = 0; c < n_chunks; ++c) { const uint32_t h = hist[c * nr + r]; hist[c * nr + r] = pos; pos += h; }
      st->col_reg_begin[r + 1] = pos;
    }
    st->col_dflows.resize_uninit(nf);
    optcc_parallel_chunks(n_chunks, nf, [&](size_t c) {
      uint32_t* pos = hist.data() + c * nr;
      const uint32_t* reg = pl->flow_region.data();
      for (uint32_t i = chunk_lo(c); i < chunk_lo(c + 1); ++i) {
        const optcc_flow_t& f = pl->flows[i];
        DFlow d;
        d.off = f.off; d.len = f.len; d.src = f.src; d.dst = f.dst; d.op = f.op;
        d.ksrc = d.kdin = d.kdout = 0; d.flags = 0; d.pad1 = 0;
        st->col_dflows[pos[reg[i]]++] = d;
      }
    });
    optcc_parallel_chunks(ncls, nf, [&](size_t c) {
      ColScratch sc;
      sc.init(in.p);
      for (uint32_t q = cls_begin[c]; q < cls_begin[c + 1]; ++q) {
        const uint32_t r = cls_regions[q];
        const uint32_t fb = st->col_reg_begin[r], fe = st->col_reg_begin[r + 1];
        if (fb == fe) { uncovered.fetch_add(1, std::memory_order_relaxed); continue; }   // no executed flow touches the region
        if (!finish_region(st->col_dflows.data() + fb, fe - fb, o, sc)) uncovered.fetch_add(1, std::memory_order_relaxed);
      }
    });
  }
  *all_covered = uncovered.load() == 0;
  // ---- 3. one work item per (region, tile) ----
  auto make_items = [&](std::vector<uint4>& items, uint64_t tu, uint64_t reserve) {
    items.clear();
    items.reserve(reserve);
    for (size_t r = 0; r < nr; ++r) {
      const uint32_t fb = st->col_reg_begin[r], fe = st->col_reg_begin[r + 1];
      if (fb == fe) continue;
      const uint64_t nunits = (pl->region_len[r] + A - 1) / A;
      for (uint64_t t = 0, ubeg = 0; ubeg < nunits; ++t, ubeg += tu)
        items.push_back(make_uint4(fb, fe, (unsigned int)t, (unsigned int)std::min<uint64_t>(nunits - ubeg, tu)));
    }
  };
  make_items(st->col_items, TU, pl->tiles_per_rank);
  if (pl->mask_tile_units != pl->tile_units) make_items(st->col_items_mask, pl->mask_tile_units, pl->mask_tiles_per_rank);
  else st->col_items_mask.clear();
}

template <int MODE>
int kernel_occupancy(int* out) {
  CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, optcc_exec_kernel<MODE>, THREADS, 0));
  return OPTCC_OK;
}

// bytes one 16-byte unit of a flow moves through HBM (what the slices are balanced on)
inline uint64_t unit_cost(const optcc_plan_t* pl, size_t i) {
  const optcc_flow_t& f = pl->flows[i];
  auto sz = [](uint8_t kind) -> uint64_t { return kind == OPTCC_KIND_F32 ? 32 : 16; };
  if (pl->kind_src.empty()) return f.op == OPTCC_OP_REDUCE ? 48 : 32;   // f32 plans
  uint64_t c = sz(pl->kind_src[i]) + sz(pl->kind_dst_out[i]);
  if (f.op == OPTCC_OP_REDUCE) c += sz(pl->kind_dst_in[i]);
  return c;
}

// Per-device launch limits (SM count, resident CTAs of every kernel instantiation), queried once per process and device.
struct DeviceLimits { int sm_count = 0, coop = 0; uint32_t max_grid = 0, max_grid_df = 0; };

int query_device_limits(int dev, DeviceLimits* out) {
  DeviceLimits lim;
  CU_TRY(cudaDeviceGetAttribute(&lim.sm_count, cudaDevAttrMultiProcessorCount, dev));
  CU_TRY(cudaDeviceGetAttribute(&lim.coop, cudaDevAttrCooperativeLaunch, dev));
  int occ = 0, o = 0, rc;
  if ((rc = kernel_occupancy<MODE_F32>(&o)) != OPTCC_OK) return rc;
  occ = o;
  if ((rc = kernel_occupancy<MODE_BF16>(&o)) != OPTCC_OK) return rc;
  occ = std::min(occ, o);
  if ((rc = kernel_occupancy<MODE_MASK1>(&o)) != OPTCC_OK) return rc;
  occ = std::min(occ, o);
  if ((rc = kernel_occupancy<MODE_MASK2>(&o)) != OPTCC_OK) return rc;
  occ = std::min(occ, o);
  if ((rc = kernel_occupancy<MODE_MASK16>(&o)) != OPTCC_OK) return rc;
  occ = std::min(occ, o);
  if ((rc = kernel_occupancy<MODE_MASK32>(&o)) != OPTCC_OK) return rc;
  occ = std::min(occ, o);
  if (occ < 1) { g_last_cuda_error = (int)cudaErrorLaunchOutOfResources; return OPTCC_ECUDA; }
  occ = std::min(occ, CTAS_PER_SM);
  lim.max_grid = std::min<uint32_t>(uint32_t(lim.sm_count) * uint32_t(occ), OPTCC_MAX_GRID);
  int od = 0;
  if ((rc = df_kernel_occupancy<MODE_F32>(&o)) != OPTCC_OK) return rc;
  od = o;
  if ((rc = df_kernel_occupancy<MODE_BF16>(&o)) != OPTCC_OK) return rc;
  od = std::min(od, o);
  if ((rc = df_kernel_occupancy<MODE_MASK1>(&o)) != OPTCC_OK) return rc;
  od = std::min(od, o);
  if ((rc = df_kernel_occupancy<MODE_MASK2>(&o)) != OPTCC_OK) return rc;
  od = std::min(od, o);
  if ((rc = df_kernel_occupancy<MODE_MASK16>(&o)) != OPTCC_OK) return rc;
  od = std::min(od, o);
  if ((rc = df_kernel_occupancy<MODE_MASK32>(&o)) != OPTCC_OK) return rc;
  od = std::min(std::min(od, o), CTAS_PER_SM);
  lim.max_grid_df = std::min<uint32_t>(uint32_t(lim.sm_count) * uint32_t(std::max(od, 0)), OPTCC_MAX_GRID);
  *out = lim;
  return OPTCC_OK;
}

int device_limits(int dev, DeviceLimits* out) {
  static std::mutex mu;
  static std::unordered_map<int, DeviceLimits> cache;
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(dev);
  if (it == cache.end()) {
    DeviceLimits lim;
    int rc = query_device_limits(dev, &lim);
    if (rc != OPTCC_OK) return rc;
    it = cache.emplace(dev, lim).first;
  }
  *out = it->second;
  return OPTCC_OK;
}

// The column executor's tables need no device: built once per plan, on the host.
int build_host_tables(optcc_plan_t* pl) {
  optcc_exec_state* st = pl->exec;
  if (!st) {
    st = new (std::nothrow) optcc_exec_state();
    if (!st) return OPTCC_ENOMEM;
    pl->exec = st;
  }
  if (st->host_built) return OPTCC_OK;
  st->column = pl->opts.exec_mode == OPTCC_EXEC_COLUMN && pl->tiles_per_rank < (uint64_t(1) << 32);
  if (st->column) {
    try {
      bool covered = false;
      build_column_state(pl, st, &covered);
      st->lazy_masks = pl->info.lazy_verify && covered;
    } catch (const std::bad_alloc&) {
      return OPTCC_ENOMEM;
    }
  }
  st->host_built = true;
  return OPTCC_OK;
}

int build_state(optcc_plan_t* pl) {
  int rc0 = build_host_tables(pl);
  if (rc0 != OPTCC_OK) return rc0;
  optcc_exec_state* st = pl->exec;
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  if (st->device == dev && st->built) return OPTCC_OK;
  st->built = false;
  st->id = g_next_id.fetch_add(1);   // new tables: every workspace must be refreshed
  st->device = dev;
  DeviceLimits lim;
  int rc = device_limits(dev, &lim);
  if (rc != OPTCC_OK) return rc;
  st->sm_count = lim.sm_count;
  st->coop = lim.coop;
  const uint32_t G = pl->opts.grid_ctas ? std::min(pl->opts.grid_ctas, lim.max_grid) : lim.max_grid;
  st->G = G;
  st->G_df = pl->opts.grid_ctas ? std::min(pl->opts.grid_ctas, lim.max_grid_df) : lim.max_grid_df;

  const optcc_plan_info_t& in = pl->info;
  const uint64_t A = in.unit_elems;
  try {
    st->built = false;
    st->df_ok = false;
    if (!st->column) {   // (column executor: region-major tables only, built by build_host_tables)
      if (in.dtype == OPTCC_BF16 && pl->kind_src.empty()) optcc_assign_kinds(pl);
      st->dflows.resize(in.n_flows);
      for (size_t i = 0; i < in.n_flows; ++i) {
        const optcc_flow_t& f = pl->flows[i];
        DFlow d;
        std::memset(&d, 0, sizeof d);
        d.off = f.off; d.len = f.len; d.src = f.src; d.dst = f.dst; d.op = f.op;
        if (!pl->kind_src.empty()) { d.ksrc = pl->kind_src[i]; d.kdin = pl->kind_dst_in[i]; d.kdout = pl->kind_dst_out[i]; }
        st->dflows[i] = d;
      }
      // dataflow tables when that executor will run; otherwise the slice table of the barrier executors
      if (pl->opts.exec_mode == OPTCC_EXEC_DATAFLOW && st->coop && st->G_df > 0) build_dataflow_tables(pl, st);
      assign_mask_flags(pl, st);
    }
    // slice table: cut every step into G slices of equal HBM bytes
    st->slices.clear();
    if (!st->df_ok && !st->column) st->slices.assign(size_t(in.n_steps) * (G + 1), Slice{0, 0, 0});
    for (uint32_t t = 0; t < in.n_steps && !st->df_ok && !st->column; ++t) {
      const uint32_t lo = pl->step_begin[t], hi = pl->step_begin[t + 1];
      uint64_t Wtot = 0;
      for (uint32_t i = lo; i < hi; ++i) Wtot += ((pl->flows[i].len + A - 1) / A) * unit_cost(pl, i);
      Slice* row = st->slices.data() + size_t(t) * (G + 1);
      uint32_t i = lo;
      uint64_t prefix = 0;  // cost of flows [lo, i)
      for (uint32_t c = 0; c <= G; ++c) {
        const uint64_t Bc = (unsigned __int128)Wtot * c / G;
        while (i < hi) {
          uint64_t w = ((pl->flows[i].len + A - 1) / A) * unit_cost(pl, i);
          if (prefix + w > Bc) break;
          prefix += w;
          ++i;
        }
        row[c].flow = i;
        row[c].pad = 0;
        row[c].unit = i < hi ? (Bc - prefix) / unit_cost(pl, i) : 0;
      }
    }
  } catch (const std::bad_alloc&) {
    return OPTCC_ENOMEM;
  }
  st->built = true;
  return OPTCC_OK;
}

int upload_tables(optcc_plan_t* pl, void* workspace, cudaStream_t stream, bool force) {
  optcc_exec_state* st = pl->exec;
  if (!force) {
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    auto it = g_ws_owner.find(workspace);
    if (it != g_ws_owner.end() && it->second == st->id) return OPTCC_OK;   // this plan's tables are already there
  }
  const optcc_ws_layout L = optcc_layout(pl);
  char* ws = static_cast<char*>(workspace);
  CU_TRY(cudaMemsetAsync(ws + L.ctrl, 0, OPTCC_CTRL_BYTES, stream));
  st->stamp_host = table_stamp(st->id);       // (a member: the copy below reads it when the stream gets there)
  CU_TRY(cudaMemcpyAsync(ws + L.ctrl + offsetof(Ctrl, stamp), &st->stamp_host, sizeof(unsigned long long), cudaMemcpyHostToDevice, stream));
  if (st->column) {
    if (!st->col_dflows.empty())
      CU_TRY(cudaMemcpyAsync(ws + L.dflows, st->col_dflows.data(), st->col_dflows.size() * sizeof(DFlow), cudaMemcpyHostToDevice, stream));
    if (!st->col_items.empty())
      CU_TRY(cudaMemcpyAsync(ws + L.col, st->col_items.data(), st->col_items.size() * sizeof(uint4), cudaMemcpyHostToDevice, stream));
    if (!st->col_items_mask.empty())
      CU_TRY(cudaMemcpyAsync(ws + L.col_mask, st->col_items_mask.data(), st->col_items_mask.size() * sizeof(uint4), cudaMemcpyHostToDevice, stream));
  } else if (!st->dflows.empty())
    CU_TRY(cudaMemcpyAsync(ws + L.dflows, st->dflows.data(), st->dflows.size() * sizeof(DFlow), cudaMemcpyHostToDevice, stream));
  if (!st->slices.empty())
    CU_TRY(cudaMemcpyAsync(ws + L.slices, st->slices.data(), st->slices.size() * sizeof(Slice), cudaMemcpyHostToDevice, stream));
  if (st->df_ok && !st->ops.empty()) {
    CU_TRY(cudaMemcpyAsync(ws + L.deps, st->deps.data(), st->deps.size() * sizeof(DDep), cudaMemcpyHostToDevice, stream));
    CU_TRY(cudaMemcpyAsync(ws + L.ops, st->ops.data(), st->ops.size() * sizeof(TileOp), cudaMemcpyHostToDevice, stream));
  }
  if (st->column && st->col_dflows.pinned()) {
    if (!st->uploaded && tl_no_cuda_alloc) {
      CU_TRY(cudaStreamSynchronize(stream));   // (optcc_execute_static creates nothing: wait for the copy instead)
    } else {
      if (!st->uploaded) CU_TRY(cudaEventCreateWithFlags(&st->uploaded, cudaEventDisableTiming));
      CU_TRY(cudaEventRecord(st->uploaded, stream));
    }
  }
  {
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    g_ws_owner[workspace] = st->id;
  }
  return OPTCC_OK;
}

inline uint32_t plan_steps(const optcc_plan_t* pl) {
  const uint32_t lim = pl->opts.step_limit;
  return lim ? std::min(lim, pl->info.n_steps) : pl->info.n_steps;
}

template <int MODE>
int launch_plan(optcc_plan_t* pl, ExecParams& P, cudaStream_t stream) {
  optcc_exec_state* st = pl->exec;
  const optcc_plan_info_t& in = pl->info;
  const uint32_t n_steps = plan_steps(pl);
  if (n_steps == 0) return OPTCC_OK;
  const bool persistent = pl->opts.exec_mode == OPTCC_EXEC_PERSISTENT && st->coop;
  const bool dataflow = pl->opts.exec_mode == OPTCC_EXEC_DATAFLOW && st->coop && st->df_ok && st->G_df > 0;
  // no silent change of executor: a device without cooperative launch (or a plan whose completion counters do not fit
  // the dataflow tables) cannot run the executor the plan names -- the caller asks for OPTCC_EXEC_PER_STEP / COLUMN itself
  if ((pl->opts.exec_mode == OPTCC_EXEC_PERSISTENT && !persistent) || (pl->opts.exec_mode == OPTCC_EXEC_DATAFLOW && !dataflow))
    return OPTCC_EUNSUPPORTED;
  if (st->column) {
    // contributor-mask runs have their own tile size (mask_tile_units) when a unit of masks is wider than 16 bytes
    const bool own_items = is_mask_mode(MODE) && !st->col_items_mask.empty();
    if (is_mask_mode(MODE)) P.col_warp = pl->mask_warp;
    if (own_items) {
      P.col_items = reinterpret_cast<const uint4*>(static_cast<char*>(static_cast<void*>(P.ctrl)) + optcc_layout(pl).col_mask);
      P.tile_units = pl->mask_tile_units;
    }
    P.col_n_items = own_items ? st->col_items_mask.size() : st->col_items.size();
    if (P.item_stride > 1)   // one shard of the items (the others run on peer GPUs, or in other calls)
      P.col_n_items = P.col_n_items > P.item_first ? (P.col_n_items - P.item_first + P.item_stride - 1) / P.item_stride : 0;
    if (P.col_n_items == 0) return OPTCC_OK;
    CU_TRY(cudaMemsetAsync(&P.ctrl->ticket, 0, sizeof(unsigned long long), stream));
    const uint32_t G = pl->opts.grid_ctas ? pl->opts.grid_ctas : uint32_t(st->sm_count) * CTAS_PER_SM;
    const unsigned int grid = (unsigned int)std::min<uint64_t>(G, P.col_n_items);
    // the stage of the bulk all-gather path: one tile (of data, or of masks: unit_elems * mask bytes per unit)
    const size_t tile_bytes = size_t(P.tile_units) * (is_mask_mode(MODE) ? size_t(in.unit_elems) * mask_bytes_of(MODE) : 16);
    P.col_stage_bytes = (unsigned int)tile_bytes;
    // partial sets are forwarded through registers when a thread's vectors are the same in every flow: one round at most
    P.mask_fwd = (is_mask_mode(MODE) && P.mask_lazy && tile_bytes / 16 <= size_t(4) * (P.col_warp ? 32 : COL_THREADS)) ? 1u : 0u;
    // f32 sums likewise (DFLOW_SRC_REG): a reduce flow adds what the flow before it stored without loading it back
    // (one-round tiles: four vectors per thread of f32; of bf16, two units per thread CTA-wide and four per lane warp-wide)
    const size_t round_units = MODE == MODE_F32 ? size_t(4) * (P.col_warp ? 32 : COL_THREADS)
                                                : (P.col_warp ? size_t(4) * 32 : size_t(2) * COL_THREADS);
    if (!is_mask_mode(MODE)) {
      P.data_fwd = (pl->opts.no_forward != 1 && P.tile_units <= round_units) ? (pl->opts.no_forward == 2 ? 1u : 3u) : 0u;
      P.mask_fwd = P.data_fwd;                          // (one switch selects the forwarding instantiation below)
    }
    constexpr bool MASKS = true;                        // every mode has a forwarding instantiation
    if (P.col_warp) {
      // warp-wide tiles: one stage per warp; a CTA's 14 warps take items on their own
      const size_t dyn = P.col_bulk ? tile_bytes * (COL_THREADS / 32) : 0;
      const unsigned int wgrid = (unsigned int)std::min<uint64_t>(G, (P.col_n_items + COL_THREADS / 32 - 1) / (COL_THREADS / 32));
      // A warp's first item is its own number, the global ticket hands out the rest: a warp that finishes early takes
      // the next tile (C3: 4.1 items per warp ran 5 static rounds, 1.47 -> 1.32 ms; C2 forced to warp-wide tiles, 131 k
      // items: 1.66 -> 1.43 ms).  Claims of several consecutive items at a time are worse than either (2 / 4 / 8 / 16 per
      // claim: C3 1.49 / 1.80 / 2.28 / 4.38 ms): neighbouring tiles must run on neighbouring warps at the same time.
      P.col_chunk = 1u;
      if (MASKS && P.mask_fwd) {
        if (dyn > 40 * 1024) CU_TRY(cudaFuncSetAttribute(optcc_wcolumn_kernel<MODE, MASKS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        optcc_wcolumn_kernel<MODE, MASKS><<<wgrid, COL_THREADS, dyn, stream>>>(P);
      } else {
        if (dyn > 40 * 1024) CU_TRY(cudaFuncSetAttribute(optcc_wcolumn_kernel<MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        optcc_wcolumn_kernel<MODE, false><<<wgrid, COL_THREADS, dyn, stream>>>(P);
      }
    } else {
      const size_t dyn = P.col_bulk ? tile_bytes : 0;
      if (MASKS && P.mask_fwd) {
        if (dyn > 40 * 1024) CU_TRY(cudaFuncSetAttribute(optcc_column_kernel<MODE, MASKS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        optcc_column_kernel<MODE, MASKS><<<grid, COL_THREADS, dyn, stream>>>(P);
      } else {
        if (dyn > 40 * 1024) CU_TRY(cudaFuncSetAttribute(optcc_column_kernel<MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        optcc_column_kernel<MODE, false><<<grid, COL_THREADS, dyn, stream>>>(P);
      }
    }
    CU_TRY(cudaGetLastError());
  } else if (dataflow) {
    P.n_ops = st->step_op_begin[n_steps];
    if (P.n_ops == 0) return OPTCC_OK;
    CU_TRY(cudaMemsetAsync(P.counters, 0, size_t(in.p) * pl->tiles_per_rank * sizeof(unsigned int), stream));
    CU_TRY(cudaMemsetAsync(&P.ctrl->ticket, 0, sizeof(unsigned long long), stream));
    void* args[] = {&P};
    const size_t dyn = P.bulk_copy ? size_t(BULK_SMEM_PER_AGENT) * DF_SLOTS : 0;
    CU_TRY(cudaLaunchCooperativeKernel((const void*)optcc_dataflow_kernel<MODE>, dim3(st->G_df), dim3(DF_THREADS), args, dyn, stream));
  } else if (persistent) {
    CU_TRY(cudaMemsetAsync(&P.ctrl->barrier, 0, sizeof(unsigned long long), stream));
    P.step_lo = 0;
    P.step_hi = n_steps;
    P.use_barrier = 1;
    void* args[] = {&P};
    CU_TRY(cudaLaunchCooperativeKernel((const void*)optcc_exec_kernel<MODE>, dim3(st->G), dim3(THREADS), args, 0, stream));
  } else {
    P.use_barrier = 0;
    for (uint32_t t = 0; t < n_steps; ++t) {
      if (pl->step_begin[t] == pl->step_begin[t + 1]) continue;
      P.step_lo = t;
      P.step_hi = t + 1;
      optcc_exec_kernel<MODE><<<st->G, THREADS, 0, stream>>>(P);
    }
    CU_TRY(cudaGetLastError());
  }
  return OPTCC_OK;
}

void fill_common(const optcc_plan_t* pl, void* workspace, ExecParams& P) {
  const optcc_ws_layout L = optcc_layout(pl);
  char* ws = static_cast<char*>(workspace);
  std::memset(&P, 0, sizeof P);
  P.flows = reinterpret_cast<const DFlow*>(ws + L.dflows);
  P.slices = reinterpret_cast<const Slice*>(ws + L.slices);
  P.ctrl = reinterpret_cast<Ctrl*>(ws + L.ctrl);
  P.shadow = reinterpret_cast<float*>(ws + L.shadow);
  P.padded_n = pl->info.padded_n;
  P.n = pl->info.n;
  P.n_ranks = pl->info.p;
  P.unit_elems = pl->info.unit_elems;
  P.deps = reinterpret_cast<const DDep*>(ws + L.deps);
  P.ops = reinterpret_cast<const TileOp*>(ws + L.ops);
  P.counters = reinterpret_cast<unsigned int*>(ws + L.counters);
  P.col_items = reinterpret_cast<const uint4*>(ws + L.col);
  P.col_n_items = 0;
  P.item_first = 0;
  P.item_stride = 1;
  P.tile_units = pl->tile_units;
  P.bulk_copy = pl->opts.copy_path == 2 ? 1u : 0u;
  P.l2_hints = 1;   // source loads evict_first, destination loads and stores evict_normal (measured best)
  // ring depth by the average tile-op size (computed once in build_state): big ops -> 2 slots (short look-ahead keeps
  // the L2 reuse distance small), small ops (small tiles, or flows shorter than a tile) -> 4 slots to hide the claim /
  // fetch / completion latency; copying agents hold their slots, so the bulk path also uses 4
  P.df_slots = (pl->exec && pl->exec->big_ops && !P.bulk_copy) ? 2 : 4;
  if (pl->opts.exec_mode == OPTCC_EXEC_COLUMN) P.l2_hints = 0;   // see optcc_column_kernel
  P.stamp = pl->exec ? table_stamp(pl->exec->id) : 0;
  P.col_pf_dist = 1; P.col_pf_l2 = 0; P.col_pf_next = 0; P.col_bulk = 1;
  P.col_bulk_policy = 1;   // bulk stores evict_first: the all-gather's results are never read again (measured: C2 1.68 -> 1.62 ms)
  P.col_warp = pl->col_warp;
  P.col_chunk = 0;
  if (pl->opts.copy_path == 1) P.col_bulk = 0;
}

}  // namespace

extern "C" int optcc_last_cuda_error(void) { return g_last_cuda_error; }

extern "C" int optcc_column_tables(optcc_plan_t* plan, const void** records, uint32_t* n_records, const void** items,
                                   uint32_t* n_items) {
  if (!plan) return OPTCC_EINVAL;
  if (plan->opts.exec_mode != OPTCC_EXEC_COLUMN) return OPTCC_EUNSUPPORTED;
  int rc = build_host_tables(plan);
  if (rc != OPTCC_OK) return rc;
  const optcc_exec_state* st = plan->exec;
  if (!st->column) return OPTCC_EUNSUPPORTED;
  if (records) *records = st->col_dflows.data();
  if (n_records) *n_records = (uint32_t)st->col_dflows.size();
  if (items) *items = st->col_items.data();
  if (n_items) *n_items = (uint32_t)st->col_items.size();
  return OPTCC_OK;
}

namespace {
int prepare_impl(optcc_plan_t* plan, void* workspace, void* stream, bool force) {
  if (!plan || !workspace || (reinterpret_cast<uintptr_t>(workspace) & 255)) return OPTCC_EINVAL;
  int rc = build_state(plan);
  if (rc != OPTCC_OK) return rc;
  return upload_tables(plan, workspace, static_cast<cudaStream_t>(stream), force);
}
}  // namespace

// Explicit call: always (re-)uploads.  optcc_execute / optcc_verify upload only if the workspace does not already
// hold this plan's tables (tracked per workspace address, so two plans may alternate on one workspace).
extern "C" int optcc_prepare(optcc_plan_t* plan, void* workspace, void* stream) {
  return prepare_impl(plan, workspace, stream, true);
}

namespace {
int execute_impl(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream_, uint32_t shard, uint32_t n_shards);
}
extern "C" int optcc_execute(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream_) {
  return execute_impl(plan, bufs, workspace, stream_, 0, 1);
}
extern "C" int optcc_execute_shard(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream_, uint32_t shard,
                                   uint32_t n_shards) {
  if (!plan || n_shards == 0 || shard >= n_shards) return OPTCC_EINVAL;
  if (n_shards > 1 && plan->opts.exec_mode != OPTCC_EXEC_COLUMN) return OPTCC_EUNSUPPORTED;   // only the column executor has independent items
  return execute_impl(plan, bufs, workspace, stream_, shard, n_shards);
}
namespace {
int execute_impl(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream_, uint32_t shard, uint32_t n_shards) {
  if (!plan || !bufs || !workspace) return OPTCC_EINVAL;
  const optcc_plan_info_t& in = plan->info;
  for (uint32_t r = 0; r < in.p; ++r)
    if (!bufs[r] || (reinterpret_cast<uintptr_t>(bufs[r]) & 15)) return OPTCC_EINVAL;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int rc = prepare_impl(plan, workspace, stream_, false);
  if (rc != OPTCC_OK) return rc;
  ExecParams P;
  fill_common(plan, workspace, P);
  if (in.p <= (uint32_t)MAX_PARAM_PTRS) {
    for (uint32_t r = 0; r < in.p; ++r) P.bufs[r] = bufs[r];
  } else {
    const optcc_ws_layout L = optcc_layout(plan);
    char* ws = static_cast<char*>(workspace);
    CU_TRY(cudaMemcpyAsync(ws + L.ptrs, bufs, size_t(in.p) * sizeof(void*), cudaMemcpyHostToDevice, stream));
    P.ptr_table = reinterpret_cast<void* const*>(ws + L.ptrs);
  }
  P.item_first = shard;
  P.item_stride = n_shards;
  return in.dtype == OPTCC_F32 ? launch_plan<MODE_F32>(plan, P, stream) : launch_plan<MODE_BF16>(plan, P, stream);
}
}  // namespace

// ---- optcc_execute_static: optcc_execute for callers that cannot allocate device memory --------------------------
// The workspace (control block, executor tables, dataflow counters, bf16 fp32 partials) is this file-scope array instead
// of caller memory.  In host code the NAME of the array is only a stand-in of the host compiler, not a device address:
// the address comes from cudaGetSymbolAddress, asked once per device with that device current, and goes to the kernels
// through ExecParams like any caller workspace.  Every GPU that loads the library holds these bytes until the process exits.
static __device__ __align__(256) unsigned char g_static_workspace[OPTCC_STATIC_WORKSPACE_BYTES];

namespace {
std::mutex g_static_mutex;
std::unordered_map<int, void*> g_static_ptr;      // device ordinal -> device address of g_static_workspace there

int static_workspace(void** out) {
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_static_mutex);
  auto it = g_static_ptr.find(dev);
  if (it == g_static_ptr.end()) {
    void* ptr = nullptr;
    CU_TRY(cudaGetSymbolAddress(&ptr, g_static_workspace));
    if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255)) return OPTCC_ECUDA;
    it = g_static_ptr.emplace(dev, ptr).first;
  }
  *out = it->second;
  return OPTCC_OK;
}
}  // namespace

extern "C" int optcc_execute_static(optcc_plan_t* plan, void* const* bufs, void* stream_) {
  if (!plan || !bufs) return OPTCC_EINVAL;
  if (plan->info.workspace_bytes > uint64_t(OPTCC_STATIC_WORKSPACE_BYTES)) return OPTCC_ETOOBIG;
  void* ws = nullptr;
  int rc = static_workspace(&ws);
  if (rc != OPTCC_OK) return rc;
  // Same path as a caller workspace from here on.  The array keeps what the last call left in it: the tables are
  // uploaded again (control block cleared, stamp rewritten) whenever the last plan to use it was another one, and every
  // launch clears its own ticket / barrier / completion counters first (launch_plan), so nothing is assumed to be zero.
  struct NoAlloc { bool was = tl_no_cuda_alloc; NoAlloc() { tl_no_cuda_alloc = true; } ~NoAlloc() { tl_no_cuda_alloc = was; } } guard;
  return optcc_execute(plan, bufs, ws, stream_);   // (tables this call has to build go to pageable host memory)
}

extern "C" int optcc_execute_host(optcc_plan_t* plan, const void* const* host_in, void* const* host_out,
                                  void* const* bufs, void* workspace, void* stream_) {
  if (!plan || !host_in || !host_out || !bufs) return OPTCC_EINVAL;
  const optcc_plan_info_t& in = plan->info;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  const size_t bytes = size_t(in.n) * (in.dtype == OPTCC_F32 ? 4 : 2);
  for (uint32_t r = 0; r < in.p; ++r) {
    if (!host_in[r] || !host_out[r] || !bufs[r]) return OPTCC_EINVAL;
    CU_TRY(cudaMemcpyAsync(bufs[r], host_in[r], bytes, cudaMemcpyHostToDevice, stream));
  }
  int rc = optcc_execute(plan, bufs, workspace, stream_);
  if (rc != OPTCC_OK) return rc;
  for (uint32_t r = 0; r < in.p; ++r) CU_TRY(cudaMemcpyAsync(host_out[r], bufs[r], bytes, cudaMemcpyDeviceToHost, stream));
  return OPTCC_OK;
}

namespace {
// The two copy streams and the events of optcc_execute_host_sharded, created on first use, one set per device.
struct ShardPipe {
  cudaStream_t in = nullptr, out = nullptr;
  cudaEvent_t begin = nullptr, end = nullptr;
  std::vector<cudaEvent_t> loaded, done;     // per shard: inputs on the device / results computed
};
std::mutex g_pipe_mutex;
std::unordered_map<int, ShardPipe> g_pipes;

int shard_pipe(int dev, size_t shards, ShardPipe** out) {
  ShardPipe& sp = g_pipes[dev];
  if (!sp.in) {
    CU_TRY(cudaStreamCreateWithFlags(&sp.in, cudaStreamNonBlocking));
    CU_TRY(cudaStreamCreateWithFlags(&sp.out, cudaStreamNonBlocking));
    CU_TRY(cudaEventCreateWithFlags(&sp.begin, cudaEventDisableTiming));
    CU_TRY(cudaEventCreateWithFlags(&sp.end, cudaEventDisableTiming));
  }
  while (sp.loaded.size() < shards) {
    cudaEvent_t a, b;
    CU_TRY(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    CU_TRY(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    sp.loaded.push_back(a);
    sp.done.push_back(b);
  }
  *out = &sp;
  return OPTCC_OK;
}
}  // namespace

namespace {
// The body of optcc_execute_host_sharded once the pipe exists: every return below leaves work queued on sp->in / sp->out
// that still reads the caller's host buffers, so the caller of this function joins those streams on any failure.
int sharded_pipeline(optcc_plan_t* plan, uint64_t shards, size_t bytes, const void* const* host_in, void* const* host_out,
                     void* const* bufs, void* workspace, void* stream_, ShardPipe* sp) {
  const optcc_plan_info_t& in = plan->info;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  CU_TRY(cudaEventRecord(sp->begin, stream));
  CU_TRY(cudaStreamWaitEvent(sp->in, sp->begin, 0));
  CU_TRY(cudaStreamWaitEvent(sp->out, sp->begin, 0));
  std::vector<void*> shard_bufs(in.p);
  for (uint64_t c = 0; c < shards; ++c) {
    const size_t o = size_t(c) * bytes;
    for (uint32_t r = 0; r < in.p; ++r)
      CU_TRY(cudaMemcpyAsync(static_cast<char*>(bufs[r]) + o, static_cast<const char*>(host_in[r]) + o, bytes,
                             cudaMemcpyHostToDevice, sp->in));
    CU_TRY(cudaEventRecord(sp->loaded[c], sp->in));
  }
  for (uint64_t c = 0; c < shards; ++c) {
    const size_t o = size_t(c) * bytes;
    for (uint32_t r = 0; r < in.p; ++r) shard_bufs[r] = static_cast<char*>(bufs[r]) + o;
    CU_TRY(cudaStreamWaitEvent(stream, sp->loaded[c], 0));
    int rc = optcc_execute(plan, shard_bufs.data(), workspace, stream_);
    if (rc != OPTCC_OK) return rc;
    CU_TRY(cudaEventRecord(sp->done[c], stream));
    CU_TRY(cudaStreamWaitEvent(sp->out, sp->done[c], 0));
    for (uint32_t r = 0; r < in.p; ++r)
      CU_TRY(cudaMemcpyAsync(static_cast<char*>(host_out[r]) + o, static_cast<char*>(bufs[r]) + o, bytes,
                             cudaMemcpyDeviceToHost, sp->out));
  }
  CU_TRY(cudaEventRecord(sp->end, sp->out));
  CU_TRY(cudaStreamWaitEvent(stream, sp->end, 0));
  return OPTCC_OK;
}
}  // namespace

extern "C" int optcc_execute_host_sharded(optcc_plan_t* plan, uint64_t n_total, const void* const* host_in,
                                          void* const* host_out, void* const* bufs, void* workspace, void* stream_) {
  if (!plan || !host_in || !host_out || !bufs || !workspace) return OPTCC_EINVAL;
  const optcc_plan_info_t& in = plan->info;
  if (n_total == 0 || n_total % in.n != 0) return OPTCC_EINVAL;
  const uint64_t shards = n_total / in.n;
  if (shards > 1 && in.n % 8 != 0) return OPTCC_EINVAL;            // shard starts stay 16-byte aligned
  if (shards > (uint64_t(1) << 16)) return OPTCC_EINVAL;
  for (uint32_t r = 0; r < in.p; ++r)
    if (!host_in[r] || !host_out[r] || !bufs[r] || (reinterpret_cast<uintptr_t>(bufs[r]) & 15)) return OPTCC_EINVAL;
  const size_t bytes = size_t(in.n) * (in.dtype == OPTCC_F32 ? 4 : 2);   // per rank and shard
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_pipe_mutex);   // one pipelined call at a time per process: the streams are shared
  ShardPipe* sp = nullptr;
  int rc = shard_pipe(dev, size_t(shards), &sp);
  if (rc != OPTCC_OK) return rc;
  rc = prepare_impl(plan, workspace, stream_, false);               // tables first, then the copies may start
  if (rc != OPTCC_OK) return rc;
  rc = sharded_pipeline(plan, shards, bytes, host_in, host_out, bufs, workspace, stream_, sp);
  if (rc != OPTCC_OK) {
    // a failed call returns only once nothing it queued can still touch host_in / host_out / bufs: the internal copy
    // streams are not the caller's to wait on (return codes ignored: the first error is the one reported)
    cudaStreamSynchronize(sp->in);
    cudaStreamSynchronize(sp->out);
    cudaStreamSynchronize(static_cast<cudaStream_t>(stream_));
  }
  return rc;
}

namespace {
int verify_impl(optcc_plan_t* plan, void* workspace, void* stream_, optcc_verify_result_t* out, uint32_t shard, uint32_t n_shards);
}
extern "C" int optcc_verify(optcc_plan_t* plan, void* workspace, void* stream_, optcc_verify_result_t* out) {
  return verify_impl(plan, workspace, stream_, out, 0, 1);
}
extern "C" int optcc_verify_shard(optcc_plan_t* plan, void* workspace, void* stream_, uint32_t shard, uint32_t n_shards,
                                  optcc_verify_result_t* out) {
  if (!plan || n_shards == 0 || shard >= n_shards) return OPTCC_EINVAL;
  if (n_shards > 1 && plan->opts.exec_mode != OPTCC_EXEC_COLUMN) return OPTCC_EUNSUPPORTED;
  return verify_impl(plan, workspace, stream_, out, shard, n_shards);
}
namespace {
int verify_impl(optcc_plan_t* plan, void* workspace, void* stream_, optcc_verify_result_t* out, uint32_t shard, uint32_t n_shards) {
  if (!plan || !workspace || !out) return OPTCC_EINVAL;
  const optcc_plan_info_t& in = plan->info;
  if (in.mask_bytes == 0) return OPTCC_EUNSUPPORTED;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int rc = prepare_impl(plan, workspace, stream_, false);
  if (rc != OPTCC_OK) return rc;
  // a shard checks the masks of its own items only: possible in the lazy form (final masks are checked by their last
  // writer); the eager form's passes run over whole arrays
  if (n_shards > 1 && !(plan->exec->column && plan->exec->lazy_masks)) return OPTCC_EUNSUPPORTED;
  const optcc_ws_layout L = optcc_layout(plan);
  char* ws = static_cast<char*>(workspace);
  char* masks = ws + L.masks;
  const uint32_t eb = in.mask_bytes;
  ExecParams P;
  fill_common(plan, workspace, P);
  for (uint32_t r = 0; r < in.p; ++r) P.bufs[r] = masks + uint64_t(r) * in.padded_n * eb;
  Ctrl init;
  std::memset(&init, 0, sizeof init);
  init.first_bad = ~0ull;
  // (counters only: the stamp and the stale count written with the tables stay as they are)
  CU_TRY(cudaMemcpyAsync(P.ctrl, &init, offsetof(Ctrl, stamp), cudaMemcpyHostToDevice, stream));
  const uint64_t vec_per_rank = in.padded_n * eb / 16;
  const unsigned int bx = (unsigned int)std::max<uint64_t>(1, std::min<uint64_t>((vec_per_rank + 1023) / 1024,
                                                          std::max<uint64_t>(1, uint64_t(plan->exec->sm_count) * 16 / in.p)));
  const dim3 blocks(bx, in.p);
  const bool lazy = plan->exec->lazy_masks;
  P.mask_lazy = lazy ? 1u : 0u;
  P.item_first = shard;
  P.item_stride = n_shards;
  if (lazy) {
    // initial masks are constants and the last writer of every range checks the final mask (assign_mask_flags); the
    // bulk-copy path would move raw memory, so the streaming warps take the copies too
    P.bulk_copy = 0;
    P.df_slots = plan->exec->big_ops ? 2 : 4;
  } else {
    optcc_mask_init_kernel<<<blocks, 256, 0, stream>>>(masks, in.padded_n, eb);
    CU_TRY(cudaGetLastError());
  }
  rc = eb == 2 ? launch_plan<MODE_MASK16>(plan, P, stream)
               : eb == 4 ? launch_plan<MODE_MASK32>(plan, P, stream)
                         : eb == 8 ? launch_plan<MODE_MASK1>(plan, P, stream) : launch_plan<MODE_MASK2>(plan, P, stream);
  if (rc != OPTCC_OK) return rc;
  if (!lazy) {
    optcc_mask_check_kernel<<<blocks, 256, 0, stream>>>(masks, in.p, in.n, in.padded_n, eb, P.ctrl);
    CU_TRY(cudaGetLastError());
  }
  Ctrl res;
  CU_TRY(cudaMemcpyAsync(&res, P.ctrl, sizeof res, cudaMemcpyDeviceToHost, stream));
  CU_TRY(cudaStreamSynchronize(stream));
  optcc_verify_result_t r;
  r.bad_elements = res.bad;
  r.overlap_elements = res.overlap;
  r.first_bad = res.first_bad;
  r.checked = uint64_t(in.p) * in.n;
  if (n_shards > 1) {   // the elements of this shard's tiles, on every rank
    const optcc_exec_state* st = plan->exec;
    const std::vector<uint4>& items = st->col_items_mask.empty() ? st->col_items : st->col_items_mask;
    const uint64_t TU = st->col_items_mask.empty() ? plan->tile_units : plan->mask_tile_units, A = in.unit_elems;
    uint64_t elems = 0;
    for (size_t i = shard; i < items.size(); i += n_shards) {
      const uint64_t len = st->col_dflows[items[i].x].len, e0 = uint64_t(items[i].z) * TU * A;
      elems += std::min<uint64_t>(uint64_t(items[i].w) * A, len - e0);
    }
    r.checked = uint64_t(in.p) * elems;
  }
  if (res.stale || res.stamp != P.stamp) return OPTCC_ESTALE;   // some launch did not find this plan's tables: nothing was verified
  *out = r;
  return (r.bad_elements || r.overlap_elements) ? OPTCC_EVERIFY : OPTCC_OK;
}
}  // namespace

// ---- buffers other processes can map (one process per GPU: optcc_execute_shard over peers' rank buffers) ----------
extern "C" int optcc_peer_alloc(uint64_t bytes, void** dev_ptr, void* handle64) {
  if (!dev_ptr || !handle64 || bytes == 0) return OPTCC_EINVAL;
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size is part of the ABI");
  void* q = nullptr;
  CU_TRY(cudaMalloc(&q, size_t(bytes)));
  cudaIpcMemHandle_t h;
  if (cudaIpcGetMemHandle(&h, q) != cudaSuccess) {
    g_last_cuda_error = (int)cudaGetLastError();
    cudaFree(q);
    return OPTCC_ECUDA;
  }
  std::memcpy(handle64, &h, 64);
  *dev_ptr = q;
  return OPTCC_OK;
}
extern "C" int optcc_peer_open(const void* handle64, void** dev_ptr) {
  if (!handle64 || !dev_ptr) return OPTCC_EINVAL;
  cudaIpcMemHandle_t h;
  std::memcpy(&h, handle64, 64);
  CU_TRY(cudaIpcOpenMemHandle(dev_ptr, h, cudaIpcMemLazyEnablePeerAccess));
  return OPTCC_OK;
}
extern "C" int optcc_peer_close(void* dev_ptr) {
  if (!dev_ptr) return OPTCC_EINVAL;
  CU_TRY(cudaIpcCloseMemHandle(dev_ptr));
  return OPTCC_OK;
}
extern "C" int optcc_peer_free(void* dev_ptr) {
  if (!dev_ptr) return OPTCC_EINVAL;
  CU_TRY(cudaFree(dev_ptr));
  return OPTCC_OK;
}

extern "C" int optcc_workspace_check(optcc_plan_t* plan, void* workspace, void* stream_) {
  if (!plan || !workspace || !plan->exec) return OPTCC_EINVAL;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  Ctrl res;
  CU_TRY(cudaMemcpyAsync(&res, static_cast<char*>(workspace) + optcc_layout(plan).ctrl, sizeof res, cudaMemcpyDeviceToHost, stream));
  CU_TRY(cudaStreamSynchronize(stream));
  return (res.stale || res.stamp != table_stamp(plan->exec->id)) ? OPTCC_ESTALE : OPTCC_OK;
}

extern "C" void optcc_workspace_forget(void* workspace) {
  std::lock_guard<std::mutex> lock(g_ws_mutex);
  g_ws_owner.erase(workspace);
}
