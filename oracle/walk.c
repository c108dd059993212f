/* TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): oracle.interpreter.run_f32 restated in plain C, so that the timed
 * CPU baseline is a compiled, multi-threaded walk of the flow table and not an interpreter number.  It shares nothing
 * with the CUDA library: the record layout is docs/PLAN_SPEC.md 3 (the oracle planner's FLOW_DTYPE), the arithmetic is
 * the paper's -- a reduce flow adds the source range into the destination range, one IEEE fp32 add per element
 * (PAPER.md:126, :132), a copy flow copies it (:130, :136) -- and the order is the table's: steps one after another
 * (:138); the flows of ONE step touch pairwise disjoint destination ranges and read nothing another flow of the step
 * writes (PLAN_SPEC 5.1, checked by oracle.interpreter.check_plan), so they are spread over the host threads.
 * Compile without contraction or reassociation: gcc -O2 -ffp-contract=off -fopenmp (oracle/cwalk.py does). */
#include <stdint.h>
#include <string.h>

typedef struct {
  uint64_t off, len;           /* elements */
  uint32_t step, seg, sec;
  uint16_t src, dst;
  uint8_t op, stage, link, part;   /* op: 0 reduce, 1 copy */
  uint32_t reserved;
} oracle_flow_t;                /* 40 bytes, packed by construction */

typedef char oracle_flow_is_40_bytes[sizeof(oracle_flow_t) == 40 ? 1 : -1];

/* y: p rows of n floats (row r = rank r's buffer), updated in place.  Returns 0, or -1 on a record out of range. */
int oracle_walk_f32(float* y, uint64_t p, uint64_t n, const oracle_flow_t* flows, const uint32_t* step_begin,
                    uint32_t n_steps) {
  int bad = 0;
  for (uint32_t t = 0; t < n_steps; ++t) {
    const int64_t lo = step_begin[t], hi = step_begin[t + 1];
#pragma omp parallel for schedule(dynamic, 1) reduction(| : bad)
    for (int64_t i = lo; i < hi; ++i) {
      const oracle_flow_t* f = flows + i;
      if (f->src >= p || f->dst >= p || f->off + f->len > n || f->step != t) { bad |= 1; continue; }
      const float* s = y + (uint64_t)f->src * n + f->off;
      float* d = y + (uint64_t)f->dst * n + f->off;
      if (f->op == 0) {
        for (uint64_t e = 0; e < f->len; ++e) d[e] = d[e] + s[e];
      } else {
        memcpy(d, s, f->len * sizeof(float));
      }
    }
  }
  return bad ? -1 : 0;
}

int oracle_walk_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
