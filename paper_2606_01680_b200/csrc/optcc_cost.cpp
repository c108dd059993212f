// alpha-beta cost model of liboptcc: modeled completion time T/T0 of a plan next to the paper's lower bounds.
//
// Event simulation under the paper's port model, as frozen in docs/PLAN_SPEC.md 6:
//   * a healthy NIC moves one element per time unit, a straggler's NIC needs ell;
//   * a NIC handles one incoming flow at a time (:124) and is full duplex: one send + one receive (:134);
//   * a transfer incident to a straggler costs ell per element (:356, :432);
//   * an NVLink lane runs at (g-1)x NIC speed per GPU and direction (:847-848, :908).
// Closed forms: T0 (:70-72), Theorems 1/2/3 (:76, :82, :112) = Table 1 (:17-26), Theorems 6/13 (:413, :664),
// Eq.(1) :173, Eq.(2) :185, D.3 :805-831, Eq.(21)/(22) :920-926.  Host only, double precision.
#include <algorithm>
#include <cmath>
#include <limits>

#include "optcc_internal.h"

extern "C" int optcc_cost(const optcc_plan_t* plan, const optcc_cost_params_t* params, optcc_cost_t* out) {
  if (!plan || !out) return OPTCC_EINVAL;
  const optcc_plan_info_t& in = plan->info;
  const double alpha = params ? params->alpha : 0.0, beta = params ? params->beta : 1.0;
  const double alat = params ? params->alpha_latency : 0.0, sync = params ? params->sync : 0.0;
  if (!(alpha >= 0.0) || !(beta > 0.0) || !std::isfinite(alpha) || !std::isfinite(beta)) return OPTCC_EINVAL;
  if (!(alat >= 0.0) || !(sync >= 0.0) || !std::isfinite(alat) || !std::isfinite(sync)) return OPTCC_EINVAL;
  const uint32_t p = in.p, g = in.g, q = in.q, m = in.m, k = in.k;
  const double n = double(in.n);

  // ---- event simulation (PLAN_SPEC 6) ----
  // per (rank, region): when its last write and its last read finish; regions = the plan's sections / P2P pieces
  struct RangeTimes { double wfin, rfin; };
  const size_t nr = plan->region_offs.size();
  std::vector<RangeTimes> rt;
  std::vector<double> send_free, recv_free;
  try {
    rt.assign(size_t(p) * nr, RangeTimes{0.0, 0.0});
    send_free.assign(size_t(p) * 2, 0.0);
    recv_free.assign(size_t(p) * 2, 0.0);
  } catch (const std::bad_alloc&) {
    return OPTCC_ENOMEM;
  }
  double T = 0.0;
  const uint32_t r_str = m ? plan->stragglers[0] * g : 0;
  double sent = 0.0, recvd = 0.0;
  const size_t nf = plan->flows.size();
  const double nv_per_elem = g > 1 ? beta / double(g - 1) : 0.0;   // NVLink lane: (g-1)x NIC speed (one division, not one per flow)
  const optcc_flow_t* const flows = plan->flows.data();
  const uint32_t* const fregion = plan->flow_region.data();
  const double* const ell = plan->ell.data();
  RangeTimes* const rtp = rt.data();
  double* const sfree = send_free.data();
  double* const rfree = recv_free.data();
  // The table lists the flows of a step by (link, stage, src, dst, off): runs of flows leave the same port one after
  // another (and often enter the same port), so a port's time is a serial (max, +) chain from flow to flow.  Both are carried
  // in registers for the length of the run (written back when the port changes) -- the loop is bound by that chain, not by memory.
  size_t cur_port = SIZE_MAX, cur_rport = SIZE_MAX;
  double sf = 0.0, rf = 0.0;
  for (size_t i = 0; i < nf; ++i) {
    const optcc_flow_t& f = flows[i];
    const size_t reg = fregion[i];
    const size_t port = size_t(f.src) * 2 + f.link;
    if (port != cur_port) {
      if (cur_port != SIZE_MAX) sfree[cur_port] = sf;
      cur_port = port;
      sf = sfree[port];
    }
    const double dur = alpha + (f.link == OPTCC_LINK_NIC ? beta * double(f.len) * std::max(ell[f.src], ell[f.dst])
                                                         : double(f.len) * nv_per_elem);
    const size_t rport = size_t(f.dst) * 2 + f.link;
    if (rport != cur_rport) {
      if (cur_rport != SIZE_MAX) rfree[cur_rport] = rf;
      cur_rport = rport;
      rf = rfree[rport];
    }
    // (region-major: the regions of a few segments are active at a time, so their p entries stay in the cache)
    RangeTimes& S = rtp[reg * p + f.src];
    RangeTimes& D = rtp[reg * p + f.dst];
    const double dep = std::max(S.wfin, std::max(D.wfin, D.rfin));   // data dependencies
    const double other = std::max(rf, dep > 0.0 ? dep + sync : 0.0);
    const double fin = std::max(sf, other) + dur;
    sf = fin;
    rf = fin;
    S.rfin = std::max(S.rfin, fin);
    D.wfin = fin + alat;                                             // usable alpha_latency after the transfer
    T = std::max(T, fin + alat);
    if (m && f.link == OPTCC_LINK_NIC) {
      if (f.src == r_str) sent += double(f.len);
      if (f.dst == r_str) recvd += double(f.len);
    }
  }
  if (cur_port != SIZE_MAX) sfree[cur_port] = sf;
  if (cur_rport != SIZE_MAX) rfree[cur_rport] = rf;

  // ---- closed forms ----
  optcc_cost_t c;
  c.T = T;
  c.T0 = beta * 2.0 * double(p - 1) * n / (double(g) * double(p));                 // :70-72 (R6: the printed q is g)
  c.T0_server = beta * 2.0 * double(q - 1) * n / (double(q) * double(g));          // base of Thm 3's series (:112, R6)
  c.T_over_T0 = T / c.T0;
  c.straggler_sent = sent;
  c.straggler_recv = recvd;
  c.reserved = 0;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  double lmax = 1.0;
  for (double l : plan->ell) lmax = std::max(lmax, l);
  c.T_ring_degraded = lmax * c.T0;   // every ring step waits for the slowest link (ICCL model, :199, :217)
  c.T_r2ccl = (g == 1 && m == 1) ? c.T0 * (1.0 + double(p) * (lmax - 1.0) / (2.0 * double(p - 1))) : nan;   // :963
  if (m == 0) {
    c.lb_table1 = c.lb_tight = c.T_closed_form = c.T_limit = c.T0;
    c.lb_table1_thm = 0; c.lb_tight_thm = 0; c.regime = 0;
  } else {
    const double l1 = plan->ell[r_str];
    if (in.construction == OPTCC_C3 && m > 1) {
      // several straggler servers with g GPUs each: E.5 (:943) gives neither bound nor time.  Every single-straggler
      // Theorem-3 bound stays valid (making the other stragglers healthy cannot slow the AllReduce down); the time form
      // composes D.3's body (:805) on n/g elements with E.4's body count k + 5.5 (:916) -- ours, not the paper's.
      const double Q = double(q), M = double(m);
      double lb = 0.0;
      for (uint32_t v : plan->stragglers) {
        const double l = plan->ell[v * g];
        lb = std::max(lb, beta * (n / g) * std::max(2.0 * l * (Q - 1.0) / (1.0 + l * (Q - 1.0)), l));
      }
      c.lb_table1 = lb;
      c.lb_tight = nan;
      c.lb_table1_thm = 3; c.lb_tight_thm = 0;
      const double ring_body = 2.0 * (Q - 1.0), str_body = l1 * (Q - M) + 2.0 * (M - 1.0);
      c.T_limit = beta * (n / g) * std::max(ring_body, str_body) / (Q - M);
      c.T_closed_form = c.T_limit * (double(k) + 5.5) / double(k);
      c.regime = str_body > ring_body ? 2 : 1;
    } else if (in.construction == OPTCC_C3) {
      const double Q = double(q);
      c.lb_table1 = beta * (n / g) * std::max(2.0 * l1 * (Q - 1.0) / (1.0 + l1 * (Q - 1.0)), l1);   // Thm 3 (:112, :538)
      c.lb_tight = beta * (n / g) * std::max(2.0 * l1 * (Q - 1.0) / (l1 * (Q - 2.0) + 2.0), l1);     // Thm 13 (:664)
      c.lb_table1_thm = 3; c.lb_tight_thm = 13;
      c.T_limit = beta * std::max(l1, 2.0) * n / g;                                                  // Eq.(21)/(22) limits
      c.T_closed_form = c.T_limit * (double(k) + 5.5) / double(k);                                   // <= (k+5.5) bodies (:916-926)
      c.regime = l1 >= 2.0 ? 2 : 1;
    } else if (m == 1) {
      const double P = double(p);
      c.lb_table1 = beta * std::max(2.0 * l1 * (P - 1.0) / (l1 * (P - 1.0) + 1.0), l1) * n;          // Thm 1 (:76)
      c.lb_tight = beta * std::max(2.0 * l1 * (P - 1.0) / (l1 * (P - 2.0) + 2.0), l1) * n;           // Thm 6 (:413)
      c.lb_table1_thm = 1; c.lb_tight_thm = 6;
      if (l1 < 2.0) {  // Eq.(2) (:185, :752): 2(p-1) l n / ((p-2) l + 2) * (k + l - 1)/k
        c.T_limit = beta * 2.0 * (P - 1.0) * l1 * n / ((P - 2.0) * l1 + 2.0);
        c.T_closed_form = c.T_limit * (double(k) + l1 - 1.0) / double(k);
        c.regime = 1;
      } else {         // Eq.(1) (:173): l n (k+1)/k
        c.T_limit = beta * l1 * n;
        c.T_closed_form = c.T_limit * (double(k) + 1.0) / double(k);
        c.regime = 2;
      }
    } else {
      double inv = 0.0;
      for (uint32_t v : plan->stragglers) inv += 1.0 / plan->ell[v * g];
      const double P = double(p), M = double(m);
      c.lb_table1 = beta * std::max(2.0 * (P - 1.0) / (P - M + inv), l1) * n;                        // Thm 2 (:82)
      c.lb_tight = nan;                                                                               // Remark 9 (:519)
      c.lb_table1_thm = 2; c.lb_tight_thm = 0;
      const double ring_body = 2.0 * (P - 1.0), str_body = l1 * (P - M) + 2.0 * (M - 1.0);            // D.3 (:805), x s
      c.T_limit = beta * std::max(ring_body, str_body) / (P - M) * n;                                 // (:831)
      c.T_closed_form = c.T_limit * (double(k) + 4.0) / double(k);                                    // (k+4) T_body (:809)
      c.regime = str_body > ring_body ? 2 : 1;
    }
  }
  if (plan->opts.ordering == 1 && in.construction == OPTCC_C1)   // one stage per body: k + 3 bodies (PLAN_SPEC C1')
    c.T_closed_form = c.T_limit * (double(k) + 3.0) / double(k);
  if (plan->opts.schedule == OPTCC_SCHED_RING_DEGRADED) {   // the baseline's own closed form; bounds stay those of the failure
    c.T_closed_form = c.T_limit = c.T_ring_degraded;
  }
  c.bodies = T * double(k) / c.T_limit;
  *out = c;
  return OPTCC_OK;
}
