// uep_oracle.cpp — CPU ORACLE for the UltraEP post-gating balance-planning path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with paper_2606_04101_b200/csrc (the CUDA
// path) and neither includes the other.
//
// Plain, slow, single-threaded C++ written from the paper (reference/PAPER.md, UltraEP):
//   O-1 histogram : Alg. 1 line 2 "Precompute lambda_e <- sum_r lambda_{r,e}"
//   O-2 plan      : Alg. 1 lines 1-25 SolveReplication, prose §5.1
//                   (PAPER.md:225-235), constraints §4.3
//   O-3 remap     : §5.2 "Token Assignment": cumulative quotas per logical
//                   expert over its physical instances, j-th token -> first instance whose
//                   cumulative quota covers j (upper-bound lookup)
//   O-4 pack      : §4.2 forward weight distribution main -> replica slot,
//                   on one GPU = a byte copy per (rank, redundant slot, tensor)
//   O-8b remap_local : §5.2 "Token Assignment" per (source rank, expert) pair
//                   over the source-wise split Q of Alg. 1 lines 26-36 (Q itself, O-8a, is
//                   computed by oracle/__init__.py::reroute_split and passed in)
//
// The planner is a heuristic (bisection over a greedy probe), so O-2 follows Algorithm 1
// step by step in the paper's order and notation; no blocking, fusion, early exit or
// reordering.  Histogram, remap and pack are plain definitions written out.
// Readings of points the paper leaves open are the ones listed in DESIGN.md §3
// (S1..S23); each is marked at the line that applies it.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): hand-worked examples A and B and the
// per-token example of the source-aware assignment (tests/golden/), the
// all-slots-to-one-expert closed form, the paper's constraints as
// invariants, numpy bincount / stable argsort, strict==tolerant at u_min=1, identity
// cases, and an exhaustive optimum bound on the tiny config.  No function here is
// "parity unpinned"; the reading S3 (rounding of tau_lo) is unpinned BY THE PAPER and is
// fixed by the worked examples only.

#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

enum { FLOOR_STRICT = 0, FLOOR_TOLERANT = 1 };

struct Transfer { int e, t, slot; int delta; };

struct Problem {
  int E, R, n_slot, u_min, beta_num, beta_den, floor_mode;
  const int32_t* lambda;          // [E]   lambda_e
  std::vector<int> home;          // [E]   h(e)
  std::vector<int64_t> ell;       // [R]   l_r = sum_{e in E_r} lambda_e
};

// Greedy feasibility probe for one threshold tau: Alg. 1 lines 6-19.
// Returns the residual excess per rank and the accepted transfers in acceptance order.
static void probe(const Problem& p, int64_t tau, std::vector<int64_t>& exc,
                  std::vector<Transfer>& accepted) {
  const int E = p.E, R = p.R;
  std::vector<int64_t> slk(R);
  std::vector<int> used(R, 0);                       // redundant slots consumed on rank t
  std::vector<std::vector<char>> hosts(E, std::vector<char>(R, 0));   // H~(e)
  exc.assign(R, 0);
  accepted.clear();
  // line 6: exc_r <- max(l_r - tau, 0), slk_r <- max(tau - l_r, 0)
  for (int r = 0; r < R; ++r) {
    exc[r] = std::max<int64_t>(p.ell[r] - tau, 0);
    slk[r] = std::max<int64_t>(tau - p.ell[r], 0);
  }
  // line 7: u~_{e,h(e)} <- lambda_e, u~_{e,t} <- 0: the temporary plan is the identity, so
  // H~(e) = {h(e)}.  (The quotas themselves are rebuilt from `accepted` by the caller.)
  for (int e = 0; e < E; ++e) hosts[e][p.home[e]] = 1;

  // line 8: foreach overloaded rank r in descending exc_r        (S5: ties -> lower rank id)
  std::vector<int> over;
  for (int r = 0; r < R; ++r) if (exc[r] > 0) over.push_back(r);
  std::stable_sort(over.begin(), over.end(), [&](int a, int b) { return exc[a] > exc[b]; });
  for (int r : over) {
    // line 9: foreach main expert e in E_r in descending lambda_e (S5: ties -> lower expert id)
    std::vector<int> mine;
    for (int e = 0; e < E; ++e) if (p.home[e] == r) mine.push_back(e);
    std::stable_sort(mine.begin(), mine.end(),
                     [&](int a, int b) { return p.lambda[a] > p.lambda[b]; });
    for (int e : mine) {
      int64_t cap = p.lambda[e];                     // line 10 (S6: cap_e = lambda_e)
      while (exc[r] > 0 && cap > 0) {                // line 11
        // line 12: T <- admissible hosts under slack, slot and no-duplicate constraints (S7)
        int t_star = -1;
        for (int t = 0; t < R; ++t) {
          if (slk[t] <= 0) continue;                 // slack
          if (used[t] >= p.n_slot) continue;         // slot budget N_slot
          if (hosts[e][t]) continue;                 // no logical expert twice on a rank
          // line 14: t* <- argmax slk_t                         (S7: ties -> lowest rank id)
          if (t_star < 0 || slk[t] > slk[t_star]) t_star = t;
        }
        if (t_star < 0) break;                       // line 13
        int64_t delta = std::min(exc[r], std::min(slk[t_star], cap));   // line 15
        if (delta < p.u_min) break;                  // line 16 (quota floor)
        // lines 17-18: move delta of e's quota from its home to t*; this creates a replica
        // in the next free redundant slot of t* (S10: slots filled 0,1,.. in accept order)
        accepted.push_back(Transfer{e, t_star, used[t_star], (int)delta});
        hosts[e][t_star] = 1;
        used[t_star] += 1;
        exc[r] -= delta; slk[t_star] -= delta; cap -= delta;            // line 19
      }
    }
  }
}

static bool feasible(const Problem& p, const std::vector<int64_t>& exc) {
  if (p.floor_mode == FLOOR_STRICT) {                // line 20 verbatim: sum_r exc_r = 0
    int64_t s = 0;
    for (int64_t x : exc) s += x;
    return s == 0;
  }
  // S8 (tolerant, default): a residual excess below the quota floor counts as drained
  for (int64_t x : exc) if (x >= p.u_min) return false;
  return true;
}

}  // namespace

extern "C" {

// ---- O-1 ------------------------------------------------------------------------------
// count[e] = |{s : ids[s] == e}| over the flat slot index s = i*k + kk; ids outside [0,E)
// are skipped and counted in *n_invalid (S14).
int uep_oracle_histogram(const int32_t* ids, int64_t S, int32_t E, int32_t* count,
                         int64_t* n_invalid) {
  for (int e = 0; e < E; ++e) count[e] = 0;
  int64_t bad = 0;
  for (int64_t s = 0; s < S; ++s) {
    int32_t e = ids[s];
    if (e < 0 || e >= E) { ++bad; continue; }
    count[e] += 1;
  }
  if (n_invalid) *n_invalid = bad;
  return 0;
}

// Static layout helpers (Table 1; S2): h(e) default floor(e*R/E);
// M = max_r |E_r| main slots per rank; main_phys[e] = index of e among E_{h(e)} ascending.
int uep_oracle_layout(int32_t E, int32_t R, const int32_t* home_in, int32_t* home_out,
                      int32_t* main_phys, int32_t* M_out) {
  std::vector<int> cnt(R, 0);
  for (int e = 0; e < E; ++e) {
    int h = home_in ? home_in[e] : (int)(((int64_t)e * R) / E);
    if (h < 0 || h >= R) return -1;
    home_out[e] = h;
    main_phys[e] = cnt[h]++;
  }
  int M = 0;
  for (int r = 0; r < R; ++r) M = std::max(M, cnt[r]);
  *M_out = M;
  return 0;
}

// ---- O-2 ------------------------------------------------------------------------------
// SolveReplication.  Outputs (caller-allocated, P = M + n_slot):
//   slot_expert[R*n_slot] X (-1 = empty)          inst_off[E+1]          CSR over experts
//   inst_rank/inst_phys/inst_cum[E + R*n_slot]    entry 0 of each expert = its main instance
//   phys_count/phys_base[R*P]                     rank_load[R]   rank_base[R+1]
//   U[E*R] dense quota table (may be NULL)
//   scalars[16]: 0 tau, 1 n_replicas, 2 max_load, 3 max_fanout (=max_e |H(e)|), 4 n_probes,
//                5 n_invalid (= S_total - sum lambda), 6 tau_lo on entry, 7 tau_hi on entry,
//                8 n_replicated_experts, rest 0
//   trace_tau/trace_feas[trace_cap]: the bisection sequence (may be NULL)
int uep_oracle_plan(const int32_t* lambda, int32_t E, int32_t R, int32_t n_slot, int32_t u_min,
                    int32_t beta_num, int32_t beta_den, int32_t floor_mode,
                    const int32_t* home_in, int64_t S_total,
                    int32_t* slot_expert, int32_t* inst_off, int32_t* inst_rank,
                    int32_t* inst_phys, int32_t* inst_cum, int32_t* phys_count,
                    int32_t* phys_base, int32_t* rank_load, int32_t* rank_base, int32_t* U,
                    int32_t* scalars, int64_t* trace_tau, int32_t* trace_feas,
                    int32_t trace_cap) {
  if (E <= 0 || R <= 0 || n_slot < 0 || u_min < 1 || beta_den <= 0 || beta_num <= 0) return -1;
  Problem p;
  p.E = E; p.R = R; p.n_slot = n_slot; p.u_min = u_min;
  p.beta_num = beta_num; p.beta_den = beta_den; p.floor_mode = floor_mode;
  p.lambda = lambda;
  p.home.resize(E);
  std::vector<int32_t> main_phys(E);
  int32_t M = 0;
  if (uep_oracle_layout(E, R, home_in, p.home.data(), main_phys.data(), &M) != 0) return -1;
  const int P = M + n_slot;

  // line 2: l_r <- sum_{e in E_r} lambda_e
  p.ell.assign(R, 0);
  int64_t S_valid = 0;
  for (int e = 0; e < E; ++e) { p.ell[p.home[e]] += lambda[e]; S_valid += lambda[e]; }

  // line 3: tau_lo <- beta * ceil((1/R) sum_r l_r), tau_hi <- max_r l_r
  // (S3: the mean is rounded up, the product with beta is truncated; all in int64)
  const int64_t mean_ceil = (S_valid + R - 1) / R;
  int64_t tau_lo = (mean_ceil * beta_num) / beta_den;
  int64_t tau_hi = 0;
  for (int r = 0; r < R; ++r) tau_hi = std::max(tau_hi, p.ell[r]);
  const int64_t tau_lo0 = tau_lo, tau_hi0 = tau_hi;

  std::vector<Transfer> best;            // U~ of the last feasible probe (S10); empty = identity (S4)
  std::vector<int64_t> exc;
  std::vector<Transfer> acc;
  int n_probes = 0;
  while (tau_lo < tau_hi) {                                  // line 4
    const int64_t tau = (tau_lo + tau_hi) / 2;               // line 5 (floor)
    probe(p, tau, exc, acc);                                 // lines 6-19
    const bool ok = feasible(p, exc);                        // line 20
    if (trace_tau && n_probes < trace_cap) { trace_tau[n_probes] = tau; trace_feas[n_probes] = ok; }
    ++n_probes;
    if (ok) { best = acc; tau_hi = tau; }                    // lines 21-22
    else    { tau_lo = tau + 1; }                            // line 24
  }
  const int64_t tau_final = tau_hi;

  // ---- materialise U~ into X, U and the cumulative reroute metadata (line 22, §5.2) ----
  std::vector<int64_t> u_main(E);
  for (int e = 0; e < E; ++e) u_main[e] = lambda[e];
  for (int i = 0; i < R * n_slot; ++i) slot_expert[i] = -1;
  for (int i = 0; i < R * P; ++i) { phys_count[i] = 0; phys_base[i] = 0; }
  if (U) for (int64_t i = 0; i < (int64_t)E * R; ++i) U[i] = 0;
  std::vector<int> n_rep(E, 0);
  for (const Transfer& x : best) {
    u_main[x.e] -= x.delta;
    n_rep[x.e] += 1;
    slot_expert[x.t * n_slot + x.slot] = x.e;                // X: x_{t,slot} = e
    phys_count[x.t * P + (M + x.slot)] = x.delta;            // redundant slot s is phys M+s
    if (U) U[(int64_t)x.e * R + x.t] += x.delta;
  }
  for (int e = 0; e < E; ++e) {
    phys_count[p.home[e] * P + main_phys[e]] = (int32_t)u_main[e];
    if (U) U[(int64_t)e * R + p.home[e]] += (int32_t)u_main[e];
  }
  // CSR: instance list of e = [main, replicas in acceptance order] (S11); inst_cum is the
  // inclusive cumulative quota ("lightweight prefix scan")
  inst_off[0] = 0;
  for (int e = 0; e < E; ++e) inst_off[e + 1] = inst_off[e] + 1 + n_rep[e];
  const int cap_inst = E + R * n_slot;
  for (int i = 0; i < cap_inst; ++i) { inst_rank[i] = -1; inst_phys[i] = -1; inst_cum[i] = 0; }
  int max_fanout = (E > 0) ? 1 : 0, n_groups = 0;
  for (int e = 0; e < E; ++e) {
    int pos = inst_off[e];
    int64_t cum = u_main[e];
    inst_rank[pos] = p.home[e]; inst_phys[pos] = main_phys[e]; inst_cum[pos] = (int32_t)cum;
    for (const Transfer& x : best) {
      if (x.e != e) continue;
      ++pos; cum += x.delta;
      inst_rank[pos] = x.t; inst_phys[pos] = M + x.slot; inst_cum[pos] = (int32_t)cum;
    }
    max_fanout = std::max(max_fanout, 1 + n_rep[e]);
    if (n_rep[e] > 0) ++n_groups;
  }
  // per-rank receive layout (S13): grouped by local physical slot, main slots first
  int64_t max_load = 0, run = 0;
  for (int r = 0; r < R; ++r) {
    int64_t b = 0;
    for (int q = 0; q < P; ++q) { phys_base[r * P + q] = (int32_t)b; b += phys_count[r * P + q]; }
    rank_load[r] = (int32_t)b;
    rank_base[r] = (int32_t)run;
    run += b;
    max_load = std::max(max_load, b);
  }
  rank_base[R] = (int32_t)run;

  for (int i = 0; i < 16; ++i) scalars[i] = 0;
  scalars[0] = (int32_t)tau_final;
  scalars[1] = (int32_t)best.size();
  scalars[2] = (int32_t)max_load;
  scalars[3] = max_fanout;
  scalars[4] = n_probes;
  scalars[5] = (int32_t)(S_total - S_valid);
  scalars[6] = (int32_t)tau_lo0;
  scalars[7] = (int32_t)tau_hi0;
  scalars[8] = n_groups;
  return 0;
}

// ---- O-3 ------------------------------------------------------------------------------
// Token assignment.  For slot s with e = ids[s]: j = #{s' < s : ids[s'] == e} (global stable
// order, S12); i = min{i : cum_i > j}; rank/phys from the CSR; offset = phys_base[rank][phys]
// + (j - cum_{i-1}) (S13); out_gate[rank_base[rank] + offset] = gate[s] as raw bytes (S17).
// Invalid ids -> (-1,-1,-1), no gate written (S14).
int uep_oracle_remap(const int32_t* ids, const void* gate, int32_t gate_bytes, int64_t S,
                     int32_t E, int32_t P, const int32_t* inst_off, const int32_t* inst_rank,
                     const int32_t* inst_phys, const int32_t* inst_cum,
                     const int32_t* phys_base, const int32_t* rank_base,
                     int32_t* out_replica, int32_t* out_rank, int32_t* out_offset,
                     void* out_gate) {
  std::vector<int64_t> seen(E, 0);
  const unsigned char* gsrc = (const unsigned char*)gate;
  unsigned char* gdst = (unsigned char*)out_gate;
  for (int64_t s = 0; s < S; ++s) {
    const int32_t e = ids[s];
    if (e < 0 || e >= E) { out_replica[s] = out_rank[s] = out_offset[s] = -1; continue; }
    const int64_t j = seen[e]++;
    int i = 0;
    const int lo = inst_off[e], n = inst_off[e + 1] - inst_off[e];
    while (i < n && !(inst_cum[lo + i] > j)) ++i;            // first instance whose cum covers j
    if (i >= n) return -2;                                   // plan does not cover the load
    const int rank = inst_rank[lo + i], phys = inst_phys[lo + i];
    const int64_t prev = (i == 0) ? 0 : inst_cum[lo + i - 1];
    const int64_t off = phys_base[rank * P + phys] + (j - prev);
    out_replica[s] = i; out_rank[s] = rank; out_offset[s] = (int32_t)off;
    if (gsrc && gdst)
      std::memcpy(gdst + (rank_base[rank] + off) * gate_bytes, gsrc + s * gate_bytes, gate_bytes);
  }
  return 0;
}

// ---- O-8b -----------------------------------------------------------------------------
// Source-aware token assignment (§5.2 "Token Assignment"): "the j-th local token
// of pair (r, e) is sent to the first physical instance whose cumulative quota covers j", the
// cumulative quotas being those of the source-wise split q[r,e,.] (Alg. 1 lines 26-36, computed
// by the caller: O-8a) in instance order.  Written as O-3 is: one pass over the slots in flat
// order, one counter per (source rank, expert) pair.
//   src(s)    = floor(i*R/T) for token i = s / k                                    (S1)
//   j         = #{s' < s : src(s') == src(s), ids[s'] == ids[s]}      (local stable rank)
//   instance  = first i with q[r][lo+0] + .. + q[r][lo+i] > j
//   offset    = phys_base[rank][phys] + sum_{r' < r} q[r'][lo+i] + (j - cumulative before i)
//               (S25: inside an instance tokens arrive by source rank, then local order)
// q: [R][inst_cap] int64, q[r][p] = q_{r,e,t} for CSR entry p of the plan (instance of e on t).
// n_inflight[r] (may be NULL) = slots of source rank r whose destination rank is not r.
int uep_oracle_remap_local(const int32_t* ids, const void* gate, int32_t gate_bytes, int64_t T,
                           int32_t k, int32_t E, int32_t R, int32_t P, int32_t inst_cap,
                           const int32_t* inst_off, const int32_t* inst_rank,
                           const int32_t* inst_phys, const int64_t* q,
                           const int32_t* phys_base, const int32_t* rank_base,
                           int32_t* out_replica, int32_t* out_rank, int32_t* out_offset,
                           void* out_gate, int32_t* n_inflight) {
  std::vector<int64_t> seen((size_t)R * E, 0);
  const unsigned char* gsrc = (const unsigned char*)gate;
  unsigned char* gdst = (unsigned char*)out_gate;
  if (n_inflight) for (int r = 0; r < R; ++r) n_inflight[r] = 0;
  for (int64_t s = 0; s < T * k; ++s) {
    const int32_t e = ids[s];
    if (e < 0 || e >= E) { out_replica[s] = out_rank[s] = out_offset[s] = -1; continue; }
    const int r = (int)(((s / k) * R) / T);                   // source rank of the token (S1)
    const int64_t j = seen[(size_t)r * E + e]++;              // j-th local token of pair (r, e)
    const int lo = inst_off[e], n = inst_off[e + 1] - inst_off[e];
    int i = 0;
    int64_t cum = 0, before = 0;
    for (; i < n; ++i) {                                      // first instance whose cumulative
      before = cum;                                           // quota of THIS source covers j
      cum += q[(size_t)r * inst_cap + lo + i];
      if (cum > j) break;
    }
    if (i >= n) return -2;                                    // split does not cover the demand
    int64_t from_lower = 0;                                   // tokens of lower source ranks come first
    for (int rr = 0; rr < r; ++rr) from_lower += q[(size_t)rr * inst_cap + lo + i];
    const int rank = inst_rank[lo + i], phys = inst_phys[lo + i];
    const int64_t off = phys_base[rank * P + phys] + from_lower + (j - before);
    out_replica[s] = i; out_rank[s] = rank; out_offset[s] = (int32_t)off;
    if (gsrc && gdst)
      std::memcpy(gdst + (rank_base[rank] + off) * gate_bytes, gsrc + s * gate_bytes, gate_bytes);
    if (n_inflight && rank != r) n_inflight[r] += 1;
  }
  return 0;
}

// ---- O-4 ------------------------------------------------------------------------------
// For every (t, s) with x_{t,s} = e != empty: dst[(t*n_slot+s)*B .. +B) = src[e*B .. +B).
// Empty slots are left untouched (S16).  One tensor per call.
int uep_oracle_pack(const int32_t* slot_expert, int32_t R, int32_t n_slot, const void* src,
                    int64_t bytes_per_expert, void* dst) {
  for (int t = 0; t < R; ++t)
    for (int s = 0; s < n_slot; ++s) {
      const int e = slot_expert[t * n_slot + s];
      if (e < 0) continue;
      std::memcpy((unsigned char*)dst + (int64_t)(t * n_slot + s) * bytes_per_expert,
                  (const unsigned char*)src + (int64_t)e * bytes_per_expert,
                  (size_t)bytes_per_expert);
    }
  return 0;
}

}  // extern "C"
