/* optcc.h -- C ABI of liboptcc: planning, costing, executing and verifying OPTCC AllReduce schedules
 * on one B200 (arxiv/paper_2606_01680, "Don't Let a Few Network Failures Slow the Entire AllReduce").
 *
 * Citations are PAPER.md:<line> (+ section / equation) and docs/PLAN_SPEC.md, which freezes the canonical
 * plan tables.  p virtual ranks' buffers live in ONE GPU's HBM; every "flow" of the paper (a section moved
 * between two ranks and either reduced into or copied over the destination) becomes a range
 * reduce / copy between two rank buffers.  No torch types, no exceptions, no CPU fallback: every entry point
 * returns an integer code; out-parameters are untouched on error.
 *
 * Pointer kinds are stated per argument: [host] = ordinary host memory, [device] = CUDA device memory of the
 * current device, [pinned] = page-locked host memory.
 */
#ifndef OPTCC_H_
#define OPTCC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OPTCC_ABI_VERSION 2
#if defined(__GNUC__)
#define OPTCC_API __attribute__((visibility("default")))
#else
#define OPTCC_API
#endif

/* element types of the rank buffers */
enum { OPTCC_F32 = 0, OPTCC_BF16 = 1 };

/* return codes */
enum {
  OPTCC_OK = 0,
  OPTCC_EINVAL = 1,       /* arguments violate PLAN_SPEC 1 (p<3 PAPER.md:68, g does not divide p, ell<1, ...) */
  OPTCC_EUNSUPPORTED = 2, /* g>1 without a straggler (NCCL's own ring); ordering 1 / ring baseline outside their
                             scope; p>128 for masks */
  OPTCC_ENOMEM = 3,
  OPTCC_ECUDA = 4,        /* a CUDA runtime call failed; optcc_last_cuda_error() has the code */
  OPTCC_EVERIFY = 5,      /* contributor-mask verification found a wrong element */
  OPTCC_ESTALE = 6,       /* the workspace did not hold this plan's tables when a kernel ran (see optcc_workspace_check) */
  OPTCC_ETOOBIG = 7       /* optcc_execute_static: the plan needs more than OPTCC_STATIC_WORKSPACE_BYTES of workspace */
};

/* PLAN_SPEC 3 enumerations */
enum { OPTCC_OP_REDUCE = 0, OPTCC_OP_COPY = 1 };
enum { OPTCC_S1 = 0, OPTCC_S2, OPTCC_S3, OPTCC_S4, OPTCC_BUB_UP, OPTCC_BUB_DOWN, OPTCC_N_COLLECT, OPTCC_N_DISTRIBUTE };
enum { OPTCC_LINK_NIC = 0, OPTCC_LINK_NVLINK = 1 };
/* constructions (PLAN_SPEC 4): C0 plain ring, C1 one straggler (4.1-4.2, App. C),
 * C2 m>=2 stragglers (App. D), C3 g>1 with one straggler server (App. E) or several (composition, E.5 :943) */
enum { OPTCC_C0 = 0, OPTCC_C1 = 1, OPTCC_C2 = 2, OPTCC_C3 = 3 };
/* schedules (PLAN_SPEC 1 option `schedule`): the baseline runs in the same executor and cost model */
enum {
  OPTCC_SCHED_OPTCC = 0,
  OPTCC_SCHED_RING_DEGRADED = 1 /* NCCL-style ring over all p ranks whatever ell is: the paper's ICCL comparison
                                   point under the bandwidth model; g must be 1 */
};
/* executor modes (opts.exec_mode).  All run the same tables and give the same bits. */
enum {
  OPTCC_EXEC_AUTO = 0,       /* the library chooses from the plan's shape (reported in optcc_plan_info_t.exec_mode): the
                                column executor, unless its work items cannot be indexed with 32 bits (then dataflow) */
  OPTCC_EXEC_PERSISTENT = 1, /* one cooperative kernel for the whole schedule, grid barrier between steps: global step
                                order, every intermediate state of the p buffers exists in memory */
  OPTCC_EXEC_PER_STEP = 2,   /* one kernel launch per step (stream order is the step barrier) */
  OPTCC_EXEC_DATAFLOW = 3,   /* one cooperative kernel, no grid barrier: every flow is cut into tiles, tile-ops are
                                claimed in table order and wait on per-(rank, range) completion counters, so a
                                tile-op starts as soon as the flows it depends on have finished there */
  OPTCC_EXEC_COLUMN = 4      /* one kernel, no synchronisation between CTAs at all: no flow ever mixes two element
                                indices (a flow moves a range rank to rank), so every dependency of :138
                                lies inside one element column.  A tile of one region is taken through every flow over
                                that region, in an order that respects those dependencies; every flow's add is carried out
                                (one IEEE operation per element, in the plan's order along the column) and the outputs are
                                bit-identical to the step-ordered executors, but there is NO global step order, and a partial
                                sum that only the next flow of the list reads and a later flow overwrites travels to that
                                flow in registers: it is not stored (opts.no_forward restores every load and store).  What
                                memory holds when the executed schedule ends -- the whole plan or its first step_limit
                                steps -- is exactly what the step-ordered executors leave: DESIGN.md 3 "what is kept, what is
                                given up" */
};

typedef struct optcc_plan optcc_plan_t; /* opaque; immutable after creation except for cached device state */

/* One flow (PLAN_SPEC 3): 40 bytes, little endian, natural alignment.  off/len in ELEMENTS. */
typedef struct optcc_flow {
  uint64_t off;      /* first element of the range (same in src and dst: a flow never moves data along n) */
  uint64_t len;      /* > 0 */
  uint32_t step;     /* steps execute in order; flows of one step are independent (PLAN_SPEC 5.1) */
  uint32_t seg;      /* segment b */
  uint32_t sec;      /* section c of the segment; 0 for bubble flows */
  uint16_t src;      /* sending rank */
  uint16_t dst;      /* receiving rank */
  uint8_t  op;       /* OPTCC_OP_* */
  uint8_t  stage;    /* OPTCC_S1.. */
  uint8_t  link;     /* OPTCC_LINK_* (cost model only) */
  uint8_t  part;     /* lambda, the leading-GPU index for g>1 */
  uint32_t reserved; /* 0 */
} optcc_flow_t;

typedef struct optcc_opts {
  uint32_t k;         /* segments; 0 = auto (PLAN_SPEC 2 "k"); else a multiple of 4 */
  uint32_t exec_mode; /* OPTCC_EXEC_*; 0 = auto */
  uint32_t grid_ctas; /* 0 = auto (SM count x resident CTAs per SM); else CTAs of the executor grid */
  uint32_t copy_path; /* copy (all-gather) tile-ops: 0 = auto (= 1, the faster one on the large configs), 1 = LDG/STG vector
                         copy by the streaming warps, 2 = cp.async.bulk (TMA 1-D) copy by the scheduler agents (dataflow only) */
  uint32_t step_limit;/* 0 = all steps; else execute / verify only the first step_limit steps (debugging and
                         profiling: a truncated schedule must FAIL verification) */
  uint32_t tile_units;/* dataflow executor: 16-byte units per tile-op; 0 = auto (224..3584: about two tile-ops per CTA and step, whole streaming rounds).
                         column executor: units per work item; 0 = auto (1792 for f32, 896 for bf16, at most the longest region) */
  uint32_t schedule;  /* OPTCC_SCHED_*: 0 = OPTCC (default), 1 = plain ring on the degraded topology (baseline) */
  uint32_t ordering;  /* stage ordering of PAPER.md:138 for one straggler, g = 1: 0 or 2 = ordering (2) S3->S1->S4->S2 (the
                         canonical plan, k+1 bodies), 1 = ordering (1) S1->S2->S3->S4 (PLAN_SPEC C1', k+3 bodies), 3 = the
                         four-pattern mix of PAPER.md:144-155 (A, C ordering (1); B, D ordering (2); PLAN_SPEC C1'', k+1 bodies) */
  uint32_t no_discard;/* 1 = keep dead source lines in L2 (disables the discard.global.L2 optimisation; for bisecting) */
  uint32_t verify_eager; /* 1 = optcc_verify initialises the mask arrays and checks them with separate passes even when
                            the plan allows the lazy form (initial masks as constants, final masks checked by their last
                            writer); same result, for bisecting.  Truncated plans (step_limit) are always eager. */
  uint32_t col_order; /* column executor, order of a region's flows: 0 = chain by chain (a flow is followed by the flow that
                         reads what it wrote; any order respecting the dependencies of PAPER.md:138 inside the column gives
                         the same bits), 1 = table order */
  uint32_t no_forward;/* column executor, data runs.  0 (default): a reduce flow whose source range is what the flow just
                         before it in the region's list produced adds that flow's registers instead of loading them back,
                         and a partial sum that is read only this way and overwritten by a later flow of the executed
                         schedule is not stored at all (it would be dropped from the caches before reaching HBM anyway).
                         1 = every flow loads both operands and stores its result; 2 = registers are forwarded but every
                         result is stored.  Same output bits in all three; 1 and 2 are for bisecting and A/B timing
                         (bench.py reports the time with 1 beside the default) */
  uint32_t reserved[4]; /* 0 */
} optcc_opts_t;

typedef struct optcc_plan_info {
  uint32_t p, g, q, m, H, k;   /* ranks, GPUs/server, servers, straggler servers, healthy servers, segments */
  uint32_t construction;       /* OPTCC_C* */
  uint32_t dtype;              /* OPTCC_F32 | OPTCC_BF16 */
  uint32_t unit_elems;         /* A = 16/sizeof(dtype) (PLAN_SPEC 2) */
  uint32_t mask_words;         /* 64-bit words a contributor mask is reported in: 1 (p<=64) or 2 (p<=128); 0 if p>128 */
  uint64_t n, n_ring, n_p2p;   /* elements per rank; on the ring path; on the P2P (bubble) path */
  uint64_t U, U_ring, U_p2p;   /* the same in 16-byte units */
  uint32_t n_steps;
  uint32_t n_flows;
  uint32_t max_flows_per_step;
  uint32_t n_sec_bounds;       /* entries of sec_bounds */
  uint32_t n_p2p_bounds;       /* entries of p2p_bounds (0 if no P2P path) */
  uint32_t mask_bytes;         /* bytes per contributor mask in the workspace: 2 (p<=16, bf16 plans), 4 (p<=32), 8 (p<=64), 16 (p<=128);
                                  0 if p>128 (optcc_verify: EUNSUPPORTED) */
  uint64_t reduce_elems;       /* sum of len over reduce flows  = (p-1) n  (Lemma 4) */
  uint64_t copy_elems;         /* sum of len over copy flows    = (p-1) n */
  uint64_t workspace_bytes;    /* device workspace optcc_execute needs (tables, barrier, bf16 fp32 partials) */
  uint64_t verify_workspace_bytes; /* device workspace optcc_verify needs (>= workspace_bytes) */
  uint64_t mask_offset_bytes;  /* after optcc_verify: the mask of (rank r, element e) is at
                                  workspace + mask_offset_bytes + (r*padded_n + e)*mask_bytes, little endian, bit i = rank i */
  uint64_t padded_n;           /* n rounded up to a multiple of 8: per-rank stride of masks and fp32 partials */
  double   plan_build_seconds; /* wall time optcc_plan spent ("< 1 ms at p=1024") */
  uint32_t lazy_verify;        /* 1: the executed steps write every (rank, section) at least once, so optcc_verify keeps
                                  the initial masks {r} as constants and lets the last writer of every range check the
                                  final mask (no initialising / checking pass over the arrays); 0: separate passes
                                  (some range keeps its initial mask, opts.verify_eager, or p > 128) */
  uint32_t exec_mode;          /* the executor this plan runs with (OPTCC_EXEC_*; never AUTO) */
} optcc_plan_info_t;

typedef struct optcc_cost_params {
  double alpha; /* fixed cost per flow that OCCUPIES its send and receive port (PAPER.md:68 excludes it: default 0) */
  double beta;  /* time per element on a healthy NIC (default 1) */
  double alpha_latency; /* latency-type fixed cost (PLAN_SPEC 6; PAPER.md:201 fn.5: about 14% of the fault-free ring's
                           time is fixed overhead): the ports are busy for the transfer only, the data is usable
                           alpha_latency later -- neighbouring windows overlap it.  Default 0 */
  double sync;  /* P2P sync message for inter-GPU dependencies: a flow that waits for data (not
                   for a port) starts `sync` after the data is usable.  Default 0 */
} optcc_cost_params_t;

typedef struct optcc_cost {
  double T;             /* completion time of the plan under the port model (PLAN_SPEC 6) */
  double T0;            /* 2(p-1)n/(g p), fault-free optimum */
  double T_over_T0;
  double T_closed_form; /* the paper's finite-k form: Eq.(1) :173 / Eq.(2) :185 (exact for C1); (k+4)T_body :809
                           and Eq.(21)/(22) :920-926 (upper bounds for C2 / C3); T0 for C0 */
  double T_limit;       /* its k -> infinity limit (:173, :185, :831, :920) */
  double lb_table1;     /* Theorem 1 (:76) / 2 (:82) / 3 (:112): the Table-1 lower bound */
  double lb_tight;      /* Theorem 6 (:413) / 13 (:664); NaN for m>1 (Remark 9, :519) */
  double T0_server;     /* 2(q-1)n/(q g): the base the Theorem-3 series are relative to */
  double bodies;        /* T / (body duration): the "(k+c)" of the finite-k factor */
  double straggler_sent;/* NIC elements sent by the slowest straggler's first GPU (z* n at the optimum, :455) */
  double straggler_recv;
  double T_ring_degraded; /* context: max(ell) * T0, the plain ring on the degraded topology (ICCL model, :199, :217) */
  double T_r2ccl;       /* context: T0 (1 + p(ell-1)/(2(p-1))), the closed form the paper plots for R2CCL (:963);
                           NaN unless g = 1 and m = 1 */
  int32_t lb_table1_thm;/* 1, 2 or 3; 0 for no straggler */
  int32_t lb_tight_thm; /* 6 or 13; 0 if none */
  int32_t regime;       /* 0 no straggler, 1 ring-bound (ell<2 resp. first max-term), 2 straggler-bound */
  int32_t reserved;
} optcc_cost_t;

typedef struct optcc_verify_result {
  uint64_t bad_elements;   /* (rank, element) pairs whose final mask is not "every rank exactly once" */
  uint64_t overlap_elements; /* (flow, element) pairs where a reduce joined overlapping contributor sets */
  uint64_t first_bad;      /* smallest r*n+e that is bad; UINT64_MAX if none */
  uint64_t checked;        /* p*n */
} optcc_verify_result_t;

/* ---- planning (host only; needs no GPU) ------------------------------------------------------------------ */

/* Build the ell-weighted stage/chunk/step plan of PAPER.md 3 (problem statement :68) and 4.1-4.4 as frozen
 * in docs/PLAN_SPEC.md.  ell [host, p doubles]: slowdown factor of every rank, >= 1; ranks of one server
 * (floor(i/g)) must share ell (PXN pooling, :274, :850).  n: elements per rank.  *out receives a new plan
 * owned by the library (optcc_plan_destroy).  Same as optcc_plan_ex with opts = NULL (k auto, executor auto). */
OPTCC_API int optcc_plan(int p, int g, const double* ell, uint64_t n, int dtype, optcc_plan_t** out);
OPTCC_API int optcc_plan_ex(int p, int g, const double* ell, uint64_t n, int dtype, const optcc_opts_t* opts,
                  optcc_plan_t** out);
/* Frees the plan's host tables.  Device state cached in a caller workspace is simply forgotten. NULL is ok. */
OPTCC_API void optcc_plan_destroy(optcc_plan_t* plan);
OPTCC_API int optcc_plan_info(const optcc_plan_t* plan, optcc_plan_info_t* out);
/* Borrowed [host] pointers, valid until optcc_plan_destroy.  Any out-pointer may be NULL.
 * flows[n_flows] sorted by (step, link, stage, src, dst, off); step_begin[n_steps+1] CSR index into it;
 * sec_bounds / p2p_bounds: section and P2P-piece boundaries in elements (PLAN_SPEC 2). */
OPTCC_API int optcc_plan_tables(const optcc_plan_t* plan, const optcc_flow_t** flows, const uint32_t** step_begin,
                      const uint64_t** sec_bounds, const uint64_t** p2p_bounds);

/* ---- alpha-beta cost model (host only) --------------------------------------------------------------------
 * Event-simulates the plan under the paper's port model (one send + one receive port per NIC, PAPER.md:124,
 * :134; ell time units per element on straggler-incident flows, :68, :356; NVLink at (g-1)x, :847, :908) and
 * reports T/T0 beside the lower bounds of Table 1 (:17-26).  params NULL = {alpha 0, beta 1}. */
OPTCC_API int optcc_cost(const optcc_plan_t* plan, const optcc_cost_params_t* params, optcc_cost_t* out);

/* ---- execution (current CUDA device) -----------------------------------------------------------------------
 * optcc_execute: in-place AllReduce.  bufs [host array of p DEVICE pointers], each n elements of the plan's
 * dtype, 16-byte aligned, pairwise disjoint.  On entry bufs[i] holds x_i; when the stream reaches the end of
 * the enqueued work every bufs[i] holds sum_j x_j and all p outputs are bitwise identical (PAPER.md:68 (ii)).
 * Every flow of the plan is carried out: the add is one IEEE operation per element, and for every element the flows that
 * touch it run in an order that respects the plan's data dependencies, so the outputs are bit-identical
 * whatever the executor.  The step-ordered and dataflow executors load both operands of every flow from memory and store
 * every destination range; the column executor keeps a partial sum in registers between two consecutive flows of a
 * column when nothing else would ever read it (OPTCC_EXEC_COLUMN, opts.no_forward).  The step-ordered executors
 * (OPTCC_EXEC_PERSISTENT / PER_STEP) additionally keep the GLOBAL step order, so every intermediate state of the p
 * buffers exists in memory; the default column executor and the dataflow executor do not (see OPTCC_EXEC_COLUMN and
 * DESIGN.md 3 "what is kept, what is given up").  With opts.step_limit = t every executor leaves exactly the state the
 * first t steps produce.
 * workspace [device, >= workspace_bytes, 256-byte aligned] owned by the caller; the first call with a given
 * workspace (or after another plan used it) builds the executor's tables on the host and uploads them; optcc_prepare
 * does this ahead of time and always re-uploads (see "Workspace contract" below).  stream: a cudaStream_t
 * (NULL = default stream).  Asynchronous: never synchronises the device or the stream; once the tables are resident
 * (after optcc_prepare or a first call) it only enqueues memsets and kernel launches (column executor: one memset
 * and one launch), so it can be captured into a CUDA graph on `stream` and replayed.
 * Errors: EINVAL (NULL / misaligned pointers), ECUDA, EUNSUPPORTED (the plan names the persistent or dataflow executor
 * and the device has no cooperative launch, or the dataflow tables do not fit 32-bit counters: the executor is never
 * changed silently -- plan_info.exec_mode is what runs). */
OPTCC_API int optcc_prepare(optcc_plan_t* plan, void* workspace, void* stream);
/* Host only, no device needed: the column executor's work list, for inspection and tests.  records [host, borrowed until
 * optcc_plan_destroy]: n_records records of 32 bytes { off u64, len u64 (elements), src u16, dst u16, op u8, ksrc u8,
 * kdin u8, kdout u8 (bf16 plans: 0 rank buffer, 1 fp32 partials), flags u32, pad u32 } -- the flows of the executed
 * steps stored region by region, inside a region in the order the executor runs them (any order that respects the data
 * dependencies of PAPER.md:138 inside the element column; opts.col_order).  items [host, borrowed]: n_items work items of
 * 16 bytes { first record, end record, tile, units in the tile } (u32 each): a tile of tile_units 16-byte units of one
 * region, taken through records [first, end).  EUNSUPPORTED unless the plan's executor is the column executor. */
OPTCC_API int optcc_column_tables(optcc_plan_t* plan, const void** records, uint32_t* n_records, const void** items,
                                  uint32_t* n_items);
OPTCC_API int optcc_execute(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream);
/* End-to-end variant: host_in [host array of p PINNED host pointers] are copied to bufs (device, as above),
 * the plan is executed, and every result is copied to host_out[i] (pinned; may equal host_in[i]).  All on
 * `stream`, asynchronous. */
OPTCC_API int optcc_execute_host(optcc_plan_t* plan, const void* const* host_in, void* const* host_out,
                       void* const* bufs, void* workspace, void* stream);
/* End-to-end, pipelined over element shards.  No flow ever mixes two element indices (the path shards along the
 * element axis), so an AllReduce of n_total elements per rank is n_total / n independent AllReduces of
 * n = plan's n elements each, all with this one plan: shard c is elements [c n, (c+1) n) of every rank.  The
 * host-to-device copy of shard c+1, the execution of shard c and the device-to-host copy of shard c-1 overlap
 * (two internal copy streams; the PCIe link carries both directions at once), so the end-to-end time approaches
 * max(H2D, D2H) instead of their sum.  host_in / host_out [host arrays of p PINNED host pointers, n_total elements
 * each]; bufs [host array of p device pointers, n_total elements each, 16-byte aligned]; workspace as for
 * optcc_execute (shards run one after another on `stream`, sharing it).  All work is ordered after what was
 * enqueued on `stream` before the call, and `stream` waits for all of it: to the caller it behaves like
 * optcc_execute_host.  The result of every shard is exactly what optcc_execute gives on that shard alone (the add
 * order per element follows the plan for n, not a plan for n_total).
 * Errors: EINVAL (NULL pointers, n_total not a multiple of n, or more than one shard with n not a multiple of 8
 * elements -- shard starts must stay 16-byte aligned), ECUDA. */
OPTCC_API int optcc_execute_host_sharded(optcc_plan_t* plan, uint64_t n_total, const void* const* host_in,
                               void* const* host_out, void* const* bufs, void* workspace, void* stream);

/* optcc_execute without a caller workspace, for callers that cannot allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the workspace is a static device array of
 * OPTCC_STATIC_WORKSPACE_BYTES inside the library (every GPU that loads the library holds it until the process exits).
 * The call itself allocates no device memory: no cudaMalloc / cudaFree / allocating library routine on any path; the
 * array's device address is looked up once per device (cudaGetSymbolAddress, on the first call with that device
 * current).  bufs, stream, the result and asynchrony are exactly optcc_execute's, whatever the plan's executor; the
 * first call with a plan (or after another plan used the array) builds the tables on the host and uploads them.
 * Limit: plans with info.workspace_bytes <= OPTCC_STATIC_WORKSPACE_BYTES (8 MiB: fp32 plans up to BASELINE config 1 =
 * C2, p = 16, n = 2^26, k = 16; bf16 plans only while their fp32 partials, 4 p n bytes, fit), else OPTCC_ETOOBIG and
 * nothing is enqueued.  ONE array per device is shared by every call and every plan and keeps the last call's
 * contents: the library re-uploads / clears what it needs, but two calls whose work overlaps on the GPU (different
 * streams without an ordering between them, or two host threads) race on it -- order them on one stream or with
 * events.  Calls through optcc_execute with a caller workspace are unaffected.
 * Errors: EINVAL, ETOOBIG, ECUDA. */
#define OPTCC_STATIC_WORKSPACE_BYTES (8u << 20)
OPTCC_API int optcc_execute_static(optcc_plan_t* plan, void* const* bufs, void* stream);

/* ---- ranks on several GPUs of one NVLink / NVSwitch domain -------------
 * One process per GPU.  Every process owns the buffers of some of the p ranks (optcc_peer_alloc: device memory plus a
 * 64-byte handle other processes can open), exchanges the handles with the others by whatever means it has (the Python
 * binding uses torch.distributed), opens theirs (optcc_peer_open) and so holds p device pointers: its own ranks' in
 * local HBM, the others' mapped over NVLink.  The path shards along the element axis (no flow mixes two element
 * indices), so G processes split the WORK ITEMS of the column executor: optcc_execute_shard(..., s, S) takes the tiles
 * i = s (mod S) of the plan through their whole flow lists exactly as optcc_execute does -- the loads of a flow whose
 * source rank lives on another GPU and the stores of a flow whose destination does are peer accesses, the transfer
 * overlaps the adds tile by tile, and there is no separate collective call.  When all S shards have run (the caller
 * joins them: stream synchronisation + a barrier among the processes) every rank buffer on every GPU holds the
 * AllReduce result, bit-identical to optcc_execute's.  Before the call every process's inputs must be in place (a
 * barrier), and nobody may touch a rank buffer until all shards are done.  shard = 0, n_shards = 1 is optcc_execute.
 * workspace: local to the calling process, as for optcc_execute.  optcc_verify_shard checks the contributor masks of
 * the shard's own tiles on arrays in the local workspace (lazy form only, else EUNSUPPORTED); `checked` counts them.
 * Errors: EINVAL (shard >= n_shards), EUNSUPPORTED (n_shards > 1 with another executor than the column executor), ECUDA.
 * Status: the host logic and the kernels run under test with two processes sharing ONE GPU (handles opened across
 * processes; tests/test_peer_shards.py); no box of this pool has a second GPU, so nothing here is measured over NVLink. */
OPTCC_API int optcc_execute_shard(optcc_plan_t* plan, void* const* bufs, void* workspace, void* stream, uint32_t shard,
                                  uint32_t n_shards);
OPTCC_API int optcc_verify_shard(optcc_plan_t* plan, void* workspace, void* stream, uint32_t shard, uint32_t n_shards,
                                 optcc_verify_result_t* out);
/* dev_ptr [out]: cudaMalloc'ed memory of `bytes` bytes on the current device; handle64 [out, host, 64 bytes]: its
 * cudaIpcMemHandle_t, valid in other processes of this machine.  optcc_peer_open maps such a handle (of ANOTHER process)
 * into the calling process; optcc_peer_close unmaps it; optcc_peer_free frees what optcc_peer_alloc returned (after
 * every peer has closed it). */
OPTCC_API int optcc_peer_alloc(uint64_t bytes, void** dev_ptr, void* handle64);
OPTCC_API int optcc_peer_open(const void* handle64, void** dev_ptr);
OPTCC_API int optcc_peer_close(void* dev_ptr);
OPTCC_API int optcc_peer_free(void* dev_ptr);

/* Workspace contract.  optcc_prepare (and the first optcc_execute / optcc_verify with a workspace) writes the plan's
 * tables AND a stamp into the workspace; the library remembers per workspace address which plan's tables it holds, so
 * later calls skip the upload.  If the caller reuses that memory for something else in between (or frees it and gets
 * the same address back from its allocator) that memory no longer holds the tables: every kernel therefore compares
 * the stamp with its own before touching a table, and a launch that finds another value does NOTHING except count
 * itself.  optcc_workspace_check synchronises `stream` and returns OPTCC_ESTALE if any launch since the last
 * optcc_prepare was such a no-op (the rank buffers are then unchanged) -- call optcc_prepare and run again;
 * optcc_verify reports the same.  optcc_workspace_forget drops the library's memory of a workspace address (call it
 * before freeing the workspace; optcc_plan_destroy forgets the workspaces of its plan). */
OPTCC_API int optcc_workspace_check(optcc_plan_t* plan, void* workspace, void* stream);
OPTCC_API void optcc_workspace_forget(void* workspace);

/* ---- verification --------------------------------------------------------------------------------------------
 * Runs the SAME step tables through the executor with contributor bitmasks as elements (rank r starts as
 * {r}; reduce = disjoint OR, copy = assign) and checks that every rank's every element ends as "all p ranks,
 * each once" (PAPER.md:68 correctness (ii)).  workspace [device, >= verify_workspace_bytes].  Synchronises
 * `stream` once to read the counters.  Returns OPTCC_EVERIFY if any element is wrong (out is still filled).
 * The masks stay in the workspace at mask_offset_bytes (see optcc_plan_info_t). */
OPTCC_API int optcc_verify(optcc_plan_t* plan, void* workspace, void* stream, optcc_verify_result_t* out);

OPTCC_API const char* optcc_strerror(int code);
OPTCC_API int optcc_last_cuda_error(void);   /* cudaError_t of the last failing CUDA call on this thread, 0 if none */
OPTCC_API int optcc_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OPTCC_H_ */
