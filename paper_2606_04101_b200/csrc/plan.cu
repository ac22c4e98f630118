// plan.cu — uep_plan: SolveReplication (Alg. 1 lines 1-25; §5.1).
//
// Latency-bound integer work (a dependent chain of arg-max steps), no HBM traffic to speak of.
// The paper's own kernel (§5.3: one CTA, state in shared memory, several
// probes across warps) is prior art; what is kept: all state on chip, one probe per warp.
// What is new:
//   * a thread-block CLUSTER of 8 CTAs shares one solve: 31+ concurrent probes on one SM queue
//     for issue slots, spread over 8 SMs each runs at the latency of its own dependent chain;
//     verdicts travel over distributed shared memory, one cluster barrier per round;
//   * per-probe state (slack, used slots) lives in REGISTERS, lane t%32 owns rank t; the
//     arg-max "largest slack, lowest rank id" is ONE redux.sync.max on a packed key
//     (slack << 8 | 255 - t); the owner is the lane whose key equals the reduced key;
//   * rank order and per-rank expert order do not depend on tau (S5): sorted once
//     into a flat visit list;
//   * the sequential bisection is reproduced exactly (S9) by speculating the next 6 levels of
//     ITS OWN tree (63 probes) and then walking the path the sequential search takes; a k-ary
//     search would not be equivalent;
//   * infeasible probes exit as soon as a visited rank keeps too much excess (S21);
//   * the no-duplicate test of Alg. 1 line 12 is provably redundant (S7: an accepted pair
//     (e,t) leaves slk_t = 0 or ends e's loop, and h(e) is overloaded hence has no slack);
//   * the probes of the LAST round log their accepted transfers, so the CTA that holds the log
//     of the final tau's probe (= U~ of the last feasible probe, S10) emits X, the CSR
//     cumulative quotas and the receive layout with all its threads; otherwise one logged
//     probe at the final tau is run (deterministic, so it reproduces that probe).
#include <algorithm>
#include <cstdlib>
#include <cstdio>
#include <cooperative_groups.h>
#include "uep_internal.cuh"

namespace uep {

namespace cg = cooperative_groups;

constexpr unsigned kFull = 0xffffffffu;
constexpr int kMaxLog = UEP_MAX_R * UEP_MAX_NSLOT;      // 1024 accepted transfers at most
constexpr int kPlanWarps = kPlanThreads / 32;
constexpr int kLogPer = kMaxLog / kPlanThreads;        // log entries handled per thread when emitting
constexpr int kEPer = UEP_MAX_E / kPlanThreads;        // experts per thread in the emit scan (blocked)
static_assert(kLogPer * kPlanThreads == kMaxLog && kEPer * kPlanThreads == UEP_MAX_E &&
              UEP_MAX_R <= kPlanThreads, "plan setup / emit: one thread per rank, kEPer experts per thread");
constexpr int kPlanLog2 = kPlanThreads == 512 ? 9 : 8;
static_assert(kPlanThreads == (1 << kPlanLog2), "rank order: threads per rank derived from log2(kPlanThreads)");
// CTAs (SMs) sharing one solve, so that the 63 probes of a round spread over many schedulers:
// 8 CTAs x 8 warps = one probe per warp, two per scheduler.  Measured on B200 (DSV3 shape): 4 / 8 /
// 16 CTAs give 22.9 / 20.6 / 20.4 us of bisection, i.e. from 8 up the probes are bound by the
// latency of their own dependent chain, not by issue slots, so the portable size 8 is used.
// A CTA has 16 warps, 8 of which probe: at ~96 registers per thread it takes 48 K of an SM's
// registers, which is deliberate — no rank_kernel / lookup_kernel CTA fits beside it, and a probe
// sharing its SM with 16-32 streaming warps runs far slower (measured: a 256-thread, 24 K-register
// version that co-resided with the rank kernel made the chain 5 us slower, 32.5 -> 37.5 us).
constexpr int kWalkWarp = kPlanWarps > 8 ? 8 : 0;   // first warp without a probe (8 probing warps per CTA)
constexpr int kPlanMaxNodes = 64;     // 2^6: six bisection levels speculated per round with 8 CTAs
constexpr int kPcSmem = 2048;                           // phys_count staged in smem if R*P fits

struct PlanSmem {
  int lam[UEP_MAX_E];
  int rexp[UEP_MAX_E];         // experts grouped by home rank, ascending id (static layout)
  int home[UEP_MAX_E];
  int main_phys[UEP_MAX_E];
  int wpos[UEP_MAX_E];         // position of e among its home rank's experts in visit order
  int u_main[UEP_MAX_E];
  int n_rep[UEP_MAX_E];
  int first[UEP_MAX_E];
  int inst_off[UEP_MAX_E + 1];
  int ell[UEP_MAX_R];
  int rload[UEP_MAX_R];
  int rpos[UEP_MAX_R];         // visit position of rank r (ranks by l_r desc, id asc)
  int roff[UEP_MAX_R + 1];
  // (padded: the probe reads one entry ahead of the one it is working on)
  int s_ell[UEP_MAX_R + 1];    // l_r in visit order
  int v_off[UEP_MAX_R + 2];    // CSR of the flat visit list: experts of the oi-th visited rank
  int v_lam[UEP_MAX_E + 1];    // lambda_e in visit order
  int v_e[UEP_MAX_E];          // expert ids in visit order
  int dscan[kMaxLog];
  int log_n[2][kPlanMaxNodes]; // accepted transfers of the probe at each tree node (per round parity)
  int node_feas[2][kPlanMaxNodes];   // probe verdict per tree node, written by its owner to every CTA
  int pc[kPcSmem];
  int pbase[kPcSmem];          // exclusive prefix of pc inside each rank (S13)
  int red_fan[kPlanWarps], red_grp[kPlanWarps];
  unsigned long long scan_tmp[kPlanWarps];
  int lo, hi, n_probes, n_log, log_buf, lo0, hi0, s_valid;
};

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int y = __shfl_up_sync(kFull, v, o);
    if (lane >= o) v += y;
  }
  return v;
}

// Block-wide inclusive scan of one 64-bit value per thread (two packed 32-bit sums), ONE barrier:
// every warp scans the kPlanWarps warp totals itself.  tmp must not be in use by another scan.
__device__ __forceinline__ unsigned long long block_incl_scan64(unsigned long long v, unsigned long long* tmp) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  unsigned long long s = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long y = __shfl_up_sync(kFull, s, o);
    if (lane >= o) s += y;
  }
  if (lane == 31) tmp[w] = s;
  __syncthreads();
  unsigned long long t = (lane < kPlanWarps) ? tmp[lane] : 0ull;
#pragma unroll
  for (int o = 1; o < kPlanWarps; o <<= 1) {
    const unsigned long long y = __shfl_up_sync(kFull, t, o);
    if (lane >= o) t += y;
  }
  const unsigned long long pre = __shfl_sync(kFull, t, (w + 31) & 31);     // total of the warps before w
  return w > 0 ? s + pre : s;
}

// One greedy feasibility probe (Alg. 1 lines 6-20) by one warp.  All control flow is
// warp-uniform.  A single warp issues one dependent instruction every ~4 cycles, so the probe is
// written for the fewest instructions on that chain: ranks and experts stream from the flat
// visit list (s_ell / v_off / v_lam, sorted once per solve), the owner of the arg-max is the lane
// whose key equals the reduced key (keys are unique: they carry the rank id), and its new key is
// the old one minus delta << 8.  LOG: also record the accepted transfers {e, t, slot, delta}.
// (Measured and dropped: keeping the top TWO keys so that the next arg-max is known without a
// reduction on the chain — the warp issues in order and ptxas consumes the reduction's uniform
// register right behind the CREDUX, so nothing overlaps: plan 15.1 -> 18.6 us.)
template <int RPL, bool LOG>
__device__ __forceinline__ bool probe(const PlanSmem& sm, const int tau, const int R,
                                      const int n_slot, const int u_min, const bool strict,
                                      const int lane, int4* __restrict__ log, int& n_log) {
  unsigned key[RPL];
  int left[RPL];                               // free redundant slots of the lane's ranks
#pragma unroll
  for (int i = 0; i < RPL; ++i) {
    const int t = lane + 32 * i;
    const int slk = (t < R) ? max(tau - sm.ell[t], 0) : 0;          // line 6
    left[i] = n_slot;
    key[i] = (slk > 0 && n_slot > 0) ? (((unsigned)slk << 8) | (unsigned)(255 - t)) : 0u;
  }
  const int brk = strict ? 1 : u_min;        // a rank is drained when exc < brk (S8)
  int nl = 0;
  // the visit list is read one entry ahead (next rank's load and list end, next expert's lambda):
  // the shared-memory latency of those loads is then off the probe's dependent chain
  int nxt_ell = sm.s_ell[0], nxt_b = sm.v_off[1], b = sm.v_off[0];
  for (int oi = 0; oi < R; ++oi) {                                  // line 8
    int exc = nxt_ell - tau;
    if (exc < brk) break;                      // ranks are sorted: every later rank is drained too
    const int a = b;
    b = nxt_b;
    nxt_ell = sm.s_ell[oi + 1];
    nxt_b = sm.v_off[oi + 2];
    int nxt_cap = sm.v_lam[a];
    bool dead = false;     // no rank can absorb u_min any more: slack only shrinks, so it stays so
    for (int ei = a; ei < b && exc >= u_min; ++ei) {                // line 9
      int cap = nxt_cap;                                            // line 10 (S6)
      nxt_cap = sm.v_lam[ei + 1];
      if (cap < u_min) break;                  // sorted by lambda: no later expert can pass line 16
      do {                                                          // line 11
        unsigned kl = key[0];
#pragma unroll
        for (int i = 1; i < RPL; ++i) kl = max(kl, key[i]);
        const unsigned km = __reduce_max_sync(kFull, kl);           // lines 12-14
        const int s = (int)(km >> 8);
        const int d = min(exc, min(s, cap));                        // line 15
        if (d < u_min) { dead = s < u_min; break; }                 // line 16 (or line 13: T empty)
        // owner lane (lines 17-19): its key becomes key - delta << 8, or 0 when the rank is full
        // (no slack or no slot left)
        const unsigned nk = (s > d) ? km - ((unsigned)d << 8) : 0u;
        int slot = 0;
#pragma unroll
        for (int i = 0; i < RPL; ++i) {
          if (key[i] == km) {
            if (LOG) slot = n_slot - left[i];
            left[i] -= 1;
            key[i] = (left[i] > 0) ? nk : 0u;
          }
        }
        if (LOG) {
          const int t = 255 - (int)(km & 255u);
          if (lane == (t & 31)) log[nl] = make_int4(sm.v_e[ei], t, slot, d);
        }
        ++nl;
        exc -= d;
        cap -= d;
      } while (min(exc, cap) > 0);
      if (dead) break;
    }
    // line 20 per rank (S21 early exit): strict needs exc == 0, tolerant exc < u_min (S8)
    if (exc >= brk) { n_log = nl; return false; }
    if (dead) {            // nothing can be moved any more: feasible iff no later rank needs to
      n_log = nl;
      return (oi + 1 >= R) || (nxt_ell - tau < brk);
    }
  }
  n_log = nl;
  return true;
}

// LOWREG (uep_plan_batched): up to four CTAs per SM at 64 registers — a single solve is slower
// that way, many solves at once are faster
template <int RPL, bool LOWREG>
__global__ void __launch_bounds__(kPlanThreads, LOWREG ? (1024 / kPlanThreads) : 1)
plan_kernel(const int32_t* __restrict__ expert_count, const int32_t* __restrict__ g_home,
            const int32_t* __restrict__ g_main_phys, const int32_t* __restrict__ g_roff,
            const int32_t* __restrict__ g_rexp, uep_plan_out out, int E, int R, int n_slot, int M,
            int P, int u_min, int beta_num, int beta_den, int strict_i, int S_total, int n_bufs,
            int log_cap, int levels, const int32_t* __restrict__ acc, int32_t* __restrict__ count_out,
            int acc_rows, int acc_pitch, int32_t* __restrict__ zero_ptr, int zero_n) {
  // acc != nullptr (uep_balance): lambda_e comes from the histogram's accumulator in the workspace
  // (acc_rows == 1), or is the column sum of the gathered count matrix Lambda[acc_rows][acc_pitch] of
  // the token-sharded path ("every rank solves the same plan" from the exchanged counts)
  // and the CTA that emits the plan also publishes it as expert_count (count_out)
  cg::cluster_group cluster = cg::this_cluster();
  const int csize = (int)cluster.num_blocks(), crank = (int)cluster.block_rank();
  // batched solve (uep_plan_batched): cluster b solves instance b; every array of instance b
  // starts b * (its element count) after instance 0's
  const int csh = 31 - __clz(csize);                 // the cluster size is a power of two (init_plan_kernels)
  const int batch_b = (int)blockIdx.x >> csh;
  expert_count += (size_t)batch_b * E;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  PlanSmem& sm = *reinterpret_cast<PlanSmem*>(smem_raw);
  // accept logs: n_bufs buffers of log_cap entries {e, t, slot, delta}; buffer 0 serves the
  // fallback probe, buffer 1+w the probe of warp w in the LAST speculation round (every probe of
  // that round is logged, so the plan normally needs no extra probe)
  int4* logs = reinterpret_cast<int4*>(smem_raw + ((sizeof(PlanSmem) + 15) & ~(size_t)15));
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool strict = strict_i != 0;

  // touch both ends of the parameter block now: the emit phase reads the plan's pointers on the
  // critical path, and a cold constant-cache line there costs several hundred cycles
  if (out.slot_expert == nullptr || out.scalars == nullptr || count_out == reinterpret_cast<int32_t*>(1)) return;
  // ---- setup, three barrier-separated phases after the wait -----------------------------------
  // the lookup kernel may start its plan-independent prologue.  Token-sharded path (acc_rows > 1): only
  // after the wait below — that prologue reads the gathered Lambda rows, which the kernels in front of
  // this one (shard_rows_kernel, the all-gather) are still writing until then
  if (acc_rows <= 1) pdl_trigger();
  // static layout first: it does not depend on the histogram (overlaps it under programmatic launch)
  for (int e = tid; e < E; e += kPlanThreads) {
    sm.home[e] = g_home[e];
    sm.main_phys[e] = g_main_phys[e];
    sm.rexp[e] = g_rexp[e];
  }
  for (int r = tid; r <= R; r += kPlanThreads) sm.roff[r] = g_roff[r];
  if (acc_rows > 1) for (int e = tid; e < E; e += kPlanThreads) sm.lam[e] = 0;
  // (token-sharded path: the per-source in-flight counters the lookup behind this kernel adds to;
  // it does so only after its own wait for this kernel, so clearing them anywhere in here is in time)
  if (blockIdx.x == 0) for (int i = tid; i < zero_n; i += kPlanThreads) zero_ptr[i] = 0;
  __syncthreads();
  pdl_wait();                      // the histogram (preceding kernel) is complete
  if (acc_rows > 1) pdl_trigger();
  // phase 1: lambda_e into shared memory, and line 2 (l_r) straight from global memory with
  // independent loads (thread r sums its own experts: no barrier between lambda and l_r)
  if (acc_rows <= 1) {
    const int32_t* lam_g = acc ? acc + 0 : expert_count;
    for (int e = tid; e < E; e += kPlanThreads) sm.lam[e] = __ldcg(lam_g + e);
    if (tid < R) {
      int s = 0;
      const int a = sm.roff[tid], b = sm.roff[tid + 1];
#pragma unroll 4
      for (int i = a; i < b; ++i) s += __ldcg(lam_g + sm.rexp[i]);
      sm.ell[tid] = s;
    }
  } else {                         // Alg. 1 line 2 in full: lambda_e = sum_r lambda_{r,e}
    // (kPlanThreads / Ecap threads per expert, each over a strided part of the rows with independent
    // loads, combined in shared memory: sm.lam was cleared before the wait)
    int ecap = 32;
    while (ecap < E) ecap <<= 1;
    const int parts = kPlanThreads / ecap, e = tid % ecap, part = tid / ecap;   // ecap <= UEP_MAX_E <= kPlanThreads
    if (e < E) {
      int s = 0;
#pragma unroll 16
      for (int r = part; r < acc_rows; r += parts) s += __ldcg(acc + (size_t)r * acc_pitch + e);
      atomicAdd(&sm.lam[e], s);
    }
    __syncthreads();
    if (tid < R) {
      int s = 0;
      for (int i = sm.roff[tid]; i < sm.roff[tid + 1]; ++i) s += sm.lam[sm.rexp[i]];
      sm.ell[tid] = s;
    }
  }
  __syncthreads();
  // phase 2
  // rank order (S5): visit position of rank r = number of ranks that come before it (l desc, id
  // asc), and in the same pass the start of its experts in the flat visit list = number of experts
  // of those ranks (no scan).  gsz threads per rank (a power of two), each over a strided part of
  // the ranks with independent loads, then a shuffle reduction inside the group.
  {
    const int gsh = min(5, kPlanLog2 - (32 - __clz(R - 1)));   // kPlanThreads >= R << gsh
    const int gsz = 1 << gsh, r = tid >> gsh, sub = tid & (gsz - 1);
    int cnt = 0, off = 0, lr = 0;
    if (r < R) {
      lr = sm.ell[r];
#pragma unroll 4
      for (int q = sub; q < R; q += gsz) {
        const int lq = sm.ell[q];
        const bool before = lq > lr || (lq == lr && q < r);
        cnt += before ? 1 : 0;
        off += before ? sm.roff[q + 1] - sm.roff[q] : 0;
      }
    }
    for (int o = gsz >> 1; o > 0; o >>= 1) {
      cnt += __shfl_xor_sync(kFull, cnt, o);
      off += __shfl_xor_sync(kFull, off, o);
    }
    if (r < R && sub == 0) { sm.rpos[r] = cnt; sm.s_ell[cnt] = lr; sm.v_off[cnt] = off; }
    if (tid == 0) { sm.s_ell[R] = 0; sm.v_off[R] = E; sm.v_off[R + 1] = E; }    // read-ahead padding
  }
  // per-rank expert order (S5): lambda desc, id asc; a thread per expert counts the experts of its
  // home rank that come before it
  for (int e = tid; e < E; e += kPlanThreads) {
    const int h = sm.home[e], le = sm.lam[e];
    const int a = sm.roff[h], b = sm.roff[h + 1];
    int cnt = 0;
#pragma unroll 4
    for (int i = a; i < b; ++i) {
      const int q = sm.rexp[i];
      const int lq = sm.lam[q];
      cnt += (lq > le || (lq == le && q < e)) ? 1 : 0;
    }
    sm.wpos[e] = cnt;
  }
  __syncthreads();
  // line 3 (S3), by the last warp alone beside the scatter below (it has no expert to place unless
  // E > kPlanThreads - 32; on every warp's path in phase 2 these two divisions cost ~950 cycles):
  // tau_lo = floor(beta * ceil(mean)), tau_hi = max l_r; S < 2^24, so 32-bit sums are exact, and
  // 32-bit divisions where the operands fit (a 64-bit division is a ~300-cycle subroutine)
  if (warp == kPlanWarps - 1) {
    int sum = 0, mx = 0;
    for (int r = lane; r < R; r += 32) { const int v = sm.ell[r]; sum += v; mx = max(mx, v); }
    sum = __reduce_add_sync(kFull, sum);
    mx = __reduce_max_sync(kFull, mx);
    const unsigned mean_ceil = ((unsigned)sum + (unsigned)R - 1u) / (unsigned)R;
    const unsigned long long prod = (unsigned long long)mean_ceil * (unsigned long long)beta_num;
    const unsigned long long tl = (prod >> 32) == 0ull ? (unsigned long long)((unsigned)prod / (unsigned)beta_den)
                                                       : prod / (unsigned long long)beta_den;
    if (lane == 0) {
      sm.lo = sm.lo0 = (int)min(tl, (unsigned long long)0x7fffffff);
      sm.hi = sm.hi0 = mx;
      sm.s_valid = sum;
      sm.n_probes = 0; sm.n_log = 0; sm.log_buf = -1;
    }
  }
  // phase 3: flat visit list (ranks in visit order, each with its experts in visit order), and the
  // emit state cleared here, off the path between the last probe and the plan's first store (no
  // probe touches it): per-expert replica counts, first log entry, staged phys_count, and by CTA 0
  // the slot map in global memory (the emitting CTA writes it after a cluster
  // barrier, or is CTA 0 itself when no round runs)
  for (int e = tid; e < E; e += kPlanThreads) {
    const int le = sm.lam[e];
    const int p = sm.v_off[sm.rpos[sm.home[e]]] + sm.wpos[e];
    sm.v_e[p] = e;
    sm.v_lam[p] = le;
    sm.u_main[e] = le; sm.n_rep[e] = 0; sm.first[e] = 0x7fffffff;
  }
  if (tid == 0) sm.v_lam[E] = 0;
  if (R * P <= kPcSmem) for (int i = tid; i < R * P; i += kPlanThreads) sm.pc[i] = 0;
  if (crank == 0) {
    int32_t* se = out.slot_expert + (size_t)batch_b * max(1, R * n_slot);
    for (int i = tid; i < R * n_slot; i += kPlanThreads) se[i] = -1;
  }
  __syncthreads();

  // ---- bisection (S9): per round up to 2^levels - 1 nodes of the SEQUENTIAL bisection tree rooted
  // at the current [lo, hi) are probed speculatively, then the path the sequential search takes is
  // walked as far as the verdicts reach.  Slot i of a round is probed by warp i / csize of CTA
  // i % csize (with 8 CTAs and 6 levels <= 2 probes per scheduler, so every probe runs at the
  // latency of its own dependent chain); the verdicts are written into EVERY CTA's shared memory
  // (DSMEM), one cluster barrier per round, every CTA walks the path redundantly.
  // WHICH nodes are speculated only decides how many rounds are needed, never the result:
  //   * first round, more than `levels` levels to go: the tree is probed where the path is
  //     expected — tau* sits at or just above tau_lo whenever the slots suffice to reach beta
  //     (every probe on the path feasible: the all-left spine).  Nodes: the complete top
  //     levels-2 levels, the spine below them, and the complete bottom levels-1 levels under
  //     the spine (every tau* in [lo, lo + 2^(levels-1)) resolves in this ONE round, any other
  //     still advances by at least levels-2 levels or to where it leaves the spine);
  //   * otherwise the complete tree of the next `levels` levels.
  // Nodes are named by their heap index in the tree rooted at [lo, hi) (1 = root, 2n = "n was
  // feasible", 2n+1 = "n was infeasible"), at any depth.
  const int n_slots = 1 << levels;
  const int top_lv = levels - 2, bot_lv = levels - 1;
  int round = 0;
  while (true) {
    const int lo = sm.lo, hi = sm.hi;
    if (lo >= hi) break;                                            // line 4
    const int buf = round & 1;
    const int depth_left = 32 - __clz(hi - lo);                     // levels on the all-feasible path
    const int bot_depth = max(depth_left - (bot_lv - 1), top_lv + 1);   // depth of the bottom subtree's root
    const int n_spine = bot_depth - 1 - top_lv;                     // spine nodes between top and bottom
    const int first_spine = 1 << top_lv, first_bot = first_spine + n_spine;
    const bool spine = round == 0 && depth_left > levels && top_lv >= 1 &&
                       first_bot + (1 << bot_lv) - 1 <= n_slots;
    // rounds whose probes may include the last feasible one log their accepted transfers
    const bool log_round = n_bufs > 1 && (spine || hi - lo < n_slots);
    auto node_of = [&](int slot) -> int {
      if (slot < 1 || slot >= n_slots) return 0;
      if (!spine || slot < first_spine) return slot;                // complete (top) levels
      if (slot < first_bot) return 1 << (top_lv + slot - first_spine);          // depth top_lv+1+k, all-left
      const int q = slot - first_bot + 1;                           // heap index inside the bottom subtree
      if (q >= (1 << bot_lv)) return 0;
      const int jl = 31 - __clz(q);
      return ((1 << (bot_depth - 1)) << jl) + (q - (1 << jl));
    };
    // the path walk below is done by the first warp that does not probe; everything of it that
    // does not need the verdicts (which node each lane stands for) is computed before the barrier
    const bool walker = warp == kWalkWarp;
    int n0 = 0, n1 = 0, d0 = 0, d1 = 0;
    bool s0 = false, s1 = false;
    if (walker) {
      n0 = node_of(lane); n1 = node_of(lane + 32);                 // lane i: the nodes of slots i and i + 32
      s0 = n0 > 0 && (n0 & (n0 - 1)) == 0; s1 = n1 > 0 && (n1 & (n1 - 1)) == 0;   // all-left nodes: powers of two
      d0 = 32 - __clz(n0); d1 = 32 - __clz(n1);                    // depth, root = 1
    }
    const int slot = warp * csize + crank;
    const int node = node_of(slot);
    if (node >= 1) {
      const int depth = 31 - __clz(node);
      int l = lo, h = hi;
      bool valid = true;
      for (int L = depth - 1; L >= 0; --L) {
        if (l >= h) { valid = false; break; }
        const int mid = (l + h) >> 1;
        if ((node >> L) & 1) l = mid + 1; else h = mid;             // 1: assumed infeasible
      }
      if (l >= h) valid = false;
      if (valid) {
        int nl = 0;
        bool f;
        if (log_round) {
          f = probe<RPL, true>(sm, (l + h) >> 1, R, n_slot, u_min, strict, lane,
                               logs + (size_t)(1 + warp) * log_cap, nl);
        } else {
          f = probe<RPL, false>(sm, (l + h) >> 1, R, n_slot, u_min, strict, lane, nullptr, nl);
        }
        if (lane < csize) {
          *cluster.map_shared_rank(&sm.node_feas[buf][slot], lane) = f ? 1 : 0;
          *cluster.map_shared_rank(&sm.log_n[buf][slot], lane) = nl;
        }
      }
    }
    if (csize > 1) cluster.sync(); else __syncthreads();
    if (walker) {
      // walk the sequential path.  A node on the path has a non-empty interval, so it was probed if
      // it was speculated at all.  (verdicts in registers: a step of the walk is two ballots, no
      // shared-memory load)
      const bool f0 = sm.node_feas[buf][lane] != 0, f1 = sm.node_feas[buf][lane + 32] != 0;
      int nd = 1, l = lo, h = hi, np = sm.n_probes, last_feas = -1;
      {
        // the run of feasible verdicts at the head of the path (usually the whole path) in one
        // step: the all-left nodes are speculated at every depth up to spine_depth, and the first
        // infeasible one ends the run
        const int spine_depth = spine ? depth_left : min(levels, depth_left);
        int dinf = spine_depth + 1;
        if (s0 && !f0) dinf = min(dinf, d0);
        if (s1 && !f1) dinf = min(dinf, d1);
        dinf = __reduce_min_sync(kFull, dinf);                       // depth of the first infeasible all-left node
        const int n_left = dinf - 1;                                 // feasible all-left nodes on the path
        h = l + ((h - l) >> n_left);                                 // lines 5, 21-22, n_left times: h <- floor((l+h)/2)
        np += n_left;
        nd = 1 << n_left;
        if (n_left > 0) {
          const unsigned m0 = __ballot_sync(kFull, s0 && d0 == n_left);
          const unsigned m1 = __ballot_sync(kFull, s1 && d1 == n_left);
          last_feas = m0 ? __ffs(m0) - 1 : 31 + __ffs(m1);
        }
      }
      while (l < h) {                                                // the rest of the path, node by node
        const bool p0 = n0 == nd, p1 = n1 == nd;
        const unsigned m = __ballot_sync(kFull, p0 || p1);
        if (m == 0u) break;                                         // not speculated: next round starts here
        const unsigned mf = __ballot_sync(kFull, (p0 && f0) || (p1 && f1));
        const int mid = (l + h) >> 1;                               // line 5
        ++np;
        if (mf) {                                                   // lines 21-22
          h = mid;
          const unsigned m0 = __ballot_sync(kFull, p0);
          last_feas = m0 ? __ffs(m0) - 1 : 31 + __ffs(m);
          nd = 2 * nd;
        } else { l = mid + 1; nd = 2 * nd + 1; }                    // line 24
      }
      if (lane == 0) {
        sm.lo = l; sm.hi = h; sm.n_probes = np;
        // the log of the last feasible probe on the path (= U~ of the final tau, S10) is usable iff
        // that probe was logged and no later logging round has reused the buffers
        if (last_feas > 0) {
          if (log_round) { sm.log_buf = last_feas; sm.n_log = sm.log_n[buf][last_feas]; }
          else sm.log_buf = -1;
        } else if (log_round) {
          sm.log_buf = -1;
        }
      }
    }
    __syncthreads();
    ++round;
  }
  const int tau = sm.hi;

  // ---- materialise (S10).  The CTA holding the log of the final tau's probe emits the plan; the
  // others are done (nothing touches their shared memory after the last cluster barrier).  If the
  // last round did not log it (the final tau was found in an earlier round, or the log buffers do
  // not fit), CTA 0 runs one logged probe at the final tau.
  const int log_node = sm.log_buf;
  const int owner = log_node < 0 ? 0 : (log_node & (csize - 1));
  if (crank != owner) return;
  const int n_probes = sm.n_probes;
  if (acc) for (int e = tid; e < E; e += kPlanThreads) count_out[e] = sm.lam[e];
  uep_plan_out o = out;            // this instance's arrays (offset only here: the probes above
  if (batch_b != 0) {              // must not carry eleven pointers in registers)
    const size_t bb = (size_t)batch_b;
    const int n_inst_cap = E + R * n_slot;
    o.slot_expert += bb * max(1, R * n_slot);
    o.inst_off += bb * (E + 1);
    o.inst_rank += bb * n_inst_cap;
    o.inst_phys += bb * n_inst_cap;
    o.inst_cum += bb * n_inst_cap;
    o.inst_base += bb * n_inst_cap;
    o.phys_count += bb * R * P;
    o.phys_base += bb * R * P;
    o.rank_load += bb * R;
    o.rank_base += bb * (R + 1);
    o.scalars += bb * UEP_N_SCALARS;
    if (o.U) o.U += bb * E * R;
  }
  const int log_buf = log_node < 0 ? 0 : 1 + (log_node >> csh);
  const int RP = R * P;
  const bool pc_in_smem = RP <= kPcSmem;
  int* pc = pc_in_smem ? sm.pc : o.phys_count;
  if (n_probes > 0 && log_node < 0) {                  // (rare; CTA-uniform condition)
    if (warp == 0) {
      int nl;
      probe<RPL, true>(sm, tau, R, n_slot, u_min, strict, lane, logs, nl);
      if (lane == 0) sm.n_log = nl;
    }
    __syncthreads();
  }
  if (!pc_in_smem || o.U) {                            // (rare: large R*P, or the dense test table)
    if (!pc_in_smem) for (int i = tid; i < RP; i += kPlanThreads) pc[i] = 0;
    if (o.U) for (int i = tid; i < E * R; i += kPlanThreads) o.U[i] = 0;
    __syncthreads();
  }
  const int4* lg = logs + (size_t)log_buf * log_cap;
  const int n_log = sm.n_log;

  // ---- emit (line 22 "materialize U~ into X" + cumulative reroute metadata, §5.2): four phases.
  // Phase A, straight from the log (thread t owns the consecutive entries t*kLogPer ..): per-expert
  // replica count / main quota / first entry, X, the replicas' phys_count and U
  if (tid == 32) {                 // everything known once the bisection has ended: off the tail of the kernel
    o.scalars[UEP_SC_TAU] = tau;
    o.scalars[UEP_SC_N_REPLICAS] = n_log;
    o.scalars[UEP_SC_N_PROBES] = n_probes;
    o.scalars[UEP_SC_N_INVALID] = S_total - sm.s_valid;
    o.scalars[UEP_SC_TAU_LO0] = sm.lo0;
    o.scalars[UEP_SC_TAU_HI0] = sm.hi0;
    for (int i = UEP_SC_N_GROUPS + 1; i < UEP_N_SCALARS; ++i) o.scalars[i] = 0;
  }
  int4 le[kLogPer];
  int dsum = 0;
#pragma unroll
  for (int j = 0; j < kLogPer; ++j) {
    const int l = tid * kLogPer + j;
    le[j] = make_int4(0, 0, 0, 0);
    if (l < n_log) {
      le[j] = lg[l];
      const int e = le[j].x, t = le[j].y, sl = le[j].z, dd = le[j].w;
      atomicSub(&sm.u_main[e], dd);
      atomicAdd(&sm.n_rep[e], 1);
      atomicMin(&sm.first[e], l);
      o.slot_expert[t * n_slot + sl] = e;                           // X
      pc[t * P + M + sl] = dd;
      if (o.U) o.U[e * R + t] = dd;
      dsum += dd;
    }
  }
  __syncthreads();
  // Phase B: one block scan for both prefix sums — instances per expert (high word; <= E + R * n_slot;
  // thread t owns the consecutive experts t*EP ..) and delta over the log (low word; <= S < 2^24, so
  // it never carries); behind it the main instances' CSR entries and, by the last warp, the receive layout
  const int EP = (E + kPlanThreads - 1) / kPlanThreads;            // 1 or 2
  int fan_mx = 0, n_grp = 0;
  {
    int v = 0;
#pragma unroll
    for (int q = 0; q < kEPer; ++q) {
      const int e = tid * EP + q;
      if (q < EP && e < E) {
        v += 1 + sm.n_rep[e];
        pc[sm.home[e] * P + sm.main_phys[e]] = sm.u_main[e];        // complete before the scan's barrier: the
      }                                                             // last warp lays out the receive buffers behind it
    }
    const unsigned long long both =
        block_incl_scan64(((unsigned long long)v << 32) | (unsigned long long)(unsigned)dsum, sm.scan_tmp);
    int pos = (int)(both >> 32) - v;
#pragma unroll
    for (int q = 0; q < kEPer; ++q) {
      const int e = tid * EP + q;
      if (q < EP && e < E) {
        const int nr = sm.n_rep[e], um = sm.u_main[e], h = sm.home[e], mp = sm.main_phys[e];
        sm.inst_off[e] = pos;
        o.inst_off[e] = pos;
        o.inst_rank[pos] = h;                                        // CSR entry of the main instance
        o.inst_phys[pos] = mp;
        o.inst_cum[pos] = um;
        if (o.U) o.U[e * R + h] = um;
        pos += 1 + nr;
        fan_mx = max(fan_mx, 1 + nr);
        n_grp += nr > 0 ? 1 : 0;
        if (e == E - 1) { sm.inst_off[E] = pos; o.inst_off[E] = pos; }
      }
    }
    int run = (int)(unsigned)both - dsum;
#pragma unroll
    for (int j = 0; j < kLogPer; ++j) {
      const int l = tid * kLogPer + j;
      run += le[j].w;
      if (l < n_log) sm.dscan[l] = run;
    }
    fan_mx = __reduce_max_sync(kFull, fan_mx);
    n_grp = __reduce_add_sync(kFull, n_grp);
    if (lane == 0) { sm.red_fan[warp] = fan_mx; sm.red_grp[warp] = n_grp; }
  }
  // receive layout (S13), an entry (rank, physical slot) per thread, handed out from the LAST thread
  // down so that it runs beside the expert threads' CSR stores: the slot's base is the sum of the
  // counts in front of it in its rank (independent loads, P - 1 at most); the thread of a rank's last
  // slot also has the rank's load.  Every phys_count was final at the scan's barrier.
  int* pbs = pc_in_smem ? sm.pbase : o.phys_base;
  for (int i = kPlanThreads - 1 - tid; i < RP; i += kPlanThreads) {
    const int r = i / P, x = i - r * P;
    int base = 0;
    for (int y = 0; y < x; ++y) base += pc[r * P + y];
    pbs[i] = base;
    if (pc_in_smem) { o.phys_base[i] = base; o.phys_count[i] = pc[i]; }
    if (x == P - 1) { const int load = base + pc[i]; o.rank_load[r] = load; sm.rload[r] = load; }
  }
  __syncthreads();
  // Phase C (last): the replicas' CSR entries (S11: acceptance order) and every instance's base
  const int* pb = pbs;                                  // bases (global ones are CTA-visible now)
#pragma unroll
  for (int j = 0; j < kLogPer; ++j) {
    const int l = tid * kLogPer + j;
    if (l < n_log) {
      const int e = le[j].x;
      const int f = sm.first[e];
      const int pos = sm.inst_off[e] + 1 + (l - f);
      const int before = (f > 0) ? sm.dscan[f - 1] : 0;
      o.inst_rank[pos] = le[j].y;
      o.inst_phys[pos] = M + le[j].z;
      o.inst_cum[pos] = sm.u_main[e] + sm.dscan[l] - before;
      o.inst_base[pos] = pb[le[j].y * P + M + le[j].z];             // S13: first token's offset in the rank's buffer
    }
  }
  for (int e = tid; e < E; e += kPlanThreads) o.inst_base[sm.inst_off[e]] = pb[sm.home[e] * P + sm.main_phys[e]];
  for (int i = E + n_log + tid; i < E + R * n_slot; i += kPlanThreads) {   // unused CSR tail
    o.inst_rank[i] = -1; o.inst_phys[i] = -1; o.inst_cum[i] = 0; o.inst_base[i] = 0;
  }
  if (warp == kPlanWarps - 1) {    // exclusive prefix over the rank loads and their maximum (lane t: ranks t*RW ..)
    const int RW = (R + 31) >> 5;
    int tot = 0, mxl = 0;
    for (int q = 0; q < RW; ++q) {
      const int r = lane * RW + q;
      if (r < R) { tot += sm.rload[r]; mxl = max(mxl, sm.rload[r]); }
    }
    const int inc = warp_incl_scan(tot, lane);
    int base = inc - tot;
    for (int q = 0; q < RW; ++q) {
      const int r = lane * RW + q;
      if (r < R) { o.rank_base[r] = base; base += sm.rload[r]; }
    }
    mxl = __reduce_max_sync(kFull, mxl);
    if (lane == 31) { o.rank_base[R] = inc; o.scalars[UEP_SC_MAX_LOAD] = mxl; }
  }
  if (tid == kPlanThreads - 64) {  // (a lane of the last warp but one)
    int max_fan = 0, n_groups = 0;
    for (int w = 0; w < kPlanWarps; ++w) { max_fan = max(max_fan, sm.red_fan[w]); n_groups += sm.red_grp[w]; }
    o.scalars[UEP_SC_MAX_FANOUT] = max_fan;
    o.scalars[UEP_SC_N_GROUPS] = n_groups;
  }
}

constexpr size_t kLogBudget = 144 * 1024;     // shared memory for the accept logs of one round (9 x 1024 entries: R = 256, N_slot = 4)

template <int RPL>
static int launch_plan_t(const Ctx* c, const int32_t* count, const uep_plan_out& plan,
                         cudaStream_t s, bool pdl, int n_inst, const int32_t* acc, int32_t* count_out,
                         int acc_rows, int acc_pitch, int32_t* zero_ptr, int zero_n) {
  const uep_config& g = c->cfg;
  const int levels = 6;                                        // 63 nodes over kPlanCluster CTAs
  const int cluster = c->plan_cluster;
  const int warps = ((1 << levels) + cluster - 1) / cluster;   // probing warps per CTA
  const int log_cap = std::max(1, g.R * g.n_slot);
  const int n_bufs = ((size_t)(1 + warps) * log_cap * sizeof(int4) <= kLogBudget) ? 1 + warps : 1;
  const size_t smem = ((sizeof(PlanSmem) + 15) & ~(size_t)15) + (size_t)n_bufs * log_cap * sizeof(int4);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(cluster * n_inst);
  cfg.blockDim = dim3(kPlanThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[3];
  int na = 0;
  attr[na].id = cudaLaunchAttributeClusterDimension;
  attr[na].val.clusterDim.x = cluster;
  attr[na].val.clusterDim.y = 1;
  attr[na].val.clusterDim.z = 1;
  ++na;
  if (pdl) {
    attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  // the planner is the critical path: when SMs free up its CTAs go before pending CTAs of the
  // kernels running beside it (uep_balance: the second wave of rank_kernel)
  // (measured, DeepSeek-V3 shape: chain 34.0 -> 32.2 us)
  attr[na].id = cudaLaunchAttributePriority;
  attr[na].val.priority = c->prio_high;
  ++na;
  cfg.attrs = attr;
  cfg.numAttrs = na;
  auto kern = n_inst > 1 ? plan_kernel<RPL, true> : plan_kernel<RPL, false>;
  UEP_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, count, (const int32_t*)c->d_home,
                                  (const int32_t*)c->d_main_phys, (const int32_t*)c->d_roff,
                                  (const int32_t*)c->d_rexp, plan, g.E, g.R, g.n_slot, c->M, c->P,
                                  g.u_min, g.beta_num, g.beta_den,
                                  g.floor_mode == UEP_FLOOR_STRICT ? 1 : 0, c->S, n_bufs, log_cap,
                                  levels, acc, count_out, acc_rows, acc_pitch, zero_ptr, zero_n));
  count_launch(c);
  return UEP_OK;
}

int launch_plan(const Ctx* c, const int32_t* count, const uep_plan_out& plan, cudaStream_t s,
                bool pdl, int n_inst, int32_t* acc, int32_t* count_out, int acc_rows, int acc_pitch,
                int32_t* zero_ptr, int zero_n) {
  const int R = c->cfg.R;
  if (n_inst <= 0) return UEP_OK;
  if (R <= 32) return launch_plan_t<1>(c, count, plan, s, pdl, n_inst, acc, count_out, acc_rows, acc_pitch, zero_ptr, zero_n);
  if (R <= 64) return launch_plan_t<2>(c, count, plan, s, pdl, n_inst, acc, count_out, acc_rows, acc_pitch, zero_ptr, zero_n);
  if (R <= 128) return launch_plan_t<4>(c, count, plan, s, pdl, n_inst, acc, count_out, acc_rows, acc_pitch, zero_ptr, zero_n);
  return launch_plan_t<8>(c, count, plan, s, pdl, n_inst, acc, count_out, acc_rows, acc_pitch, zero_ptr, zero_n);
}

template <int RPL>
static int init_plan_one(int& max16) {
  const int bytes = (int)(sizeof(PlanSmem) + 16 + kLogBudget);
  UEP_CUDA_TRY(cudaFuncSetAttribute(plan_kernel<RPL, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(plan_kernel<RPL, false>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  UEP_CUDA_TRY(cudaFuncSetAttribute(plan_kernel<RPL, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(plan_kernel<RPL, true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  if (prefer_max_smem(plan_kernel<RPL, false>) != UEP_OK || prefer_max_smem(plan_kernel<RPL, true>) != UEP_OK) return UEP_ERR_CUDA;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(16);
  cfg.blockDim = dim3(kPlanThreads);
  cfg.dynamicSmemBytes = bytes;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 16;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, plan_kernel<RPL, false>, &cfg) != cudaSuccess) { cudaGetLastError(); n = 0; }
  max16 = std::min(max16, n);
  return UEP_OK;
}

int init_plan_kernels(Ctx* c) {
  int max16 = 1 << 30;
  int rc = init_plan_one<1>(max16);
  if (rc == UEP_OK) rc = init_plan_one<2>(max16);
  if (rc == UEP_OK) rc = init_plan_one<4>(max16);
  if (rc == UEP_OK) rc = init_plan_one<8>(max16);
  // 8 CTAs x 8 probing warps cover the 64 tree slots of a round (launch_plan_t: levels = 6); the
  // path walk relies on every speculated slot having an owner, so the size is not configurable.
  // (The verdict table is deliberately NOT cleared during setup: a peer CTA whose probe exits
  // early may already have written its verdict into this CTA's shared memory by then.)
  c->plan_cluster = 8;
  static_assert(8 * 8 >= kPlanMaxNodes, "every tree slot of a round needs a probing warp");
  (void)max16;
  return rc;
}

}  // namespace uep
