// remap.cu — uep_remap: token assignment (§5.2 "Token Assignment").
//
// For slot s with expert e: j = global stable rank of s among the slots of e; instance
// i = first whose cumulative quota exceeds j (upper-bound lookup); destination
// (rank, offset) inside that rank's receive buffer; gate copied bit-exact (moved as raw
// 16/32-bit integers, S17).
//
// HBM-bound: 4 B id + g B gate read, 12 B + g B written per slot (24 B/slot for fp32 gates).
// It is a stable 512-bin multi-split.  One CTA per chunk; every warp owns a contiguous span of
// the chunk and loads all its ids and gates up front (coalesced 128 B per warp-load).  While
// those loads fly, the CTA sums the rows of the chunk table below its own (its base rank per
// expert, one round of independent int4 L2 loads) and stages the plan's CSR in shared memory.
// Ranking inside a warp: the peer mask of a lane (lanes holding the same expert) is the AND of
// NB ballots, one per bit of the expert id — independent instructions that pipeline, unlike
// match.any; the lowest peer adds the group size to a warp-private counter row and the old
// value is shuffled to its peers.  One cross-warp scan per expert column then gives the
// CTA-wide stable rank.  The order is fixed by construction (no order-dependent atomics).
// Lookup: per CTA and expert the instance holding the CTA's first slot is found once; a slot
// advances from there (0 or 1 steps in practice: a CTA's window rarely crosses a quota edge).
#include "uep_internal.cuh"

namespace uep {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr int kMaxInst = UEP_MAX_E + UEP_MAX_R * UEP_MAX_NSLOT;   // 1536 CSR entries at most

// dynamic shared memory layout (ints)
struct RemapSmem {
  int *cnt, *base, *s_off, *first, *rbase, *i_cum, *i_dbase, *i_gbase, *i_rank;
};
__host__ __device__ inline size_t remap_cnt_ints(int E_pad) {
  const size_t a = (size_t)kRemapWarps * E_pad;
  return a > (size_t)kColPartInts ? a : (size_t)kColPartInts;    // also the column-sum scratch
}
__host__ __device__ inline size_t remap_smem_ints(int E_pad, int R, int inst_cap) {
  return remap_cnt_ints(E_pad) + E_pad + (E_pad + 4) + E_pad + (R + 4) + 4 * (size_t)inst_cap;
}

template <typename GateT, int NB>
__global__ void __launch_bounds__(kRemapThreads, 1)
remap_kernel(const int32_t* __restrict__ ids, const GateT* __restrict__ gate, int S, int E,
             int E_pad, int R, int inst_cap, int chunk_len, const int32_t* __restrict__ table,
             const int32_t* __restrict__ g_inst_off, const int32_t* __restrict__ g_inst_rank,
             const int32_t* __restrict__ g_inst_cum, const int32_t* __restrict__ g_inst_base,
             const int32_t* __restrict__ g_rank_base, int32_t* __restrict__ out_replica,
             int32_t* __restrict__ out_rank, int32_t* __restrict__ out_offset,
             GateT* __restrict__ out_gate) {
  extern __shared__ __align__(16) int smem[];
  int* cnt = smem;                               // [warps][E_pad]; scratch of column_sums first
  int* base = cnt + remap_cnt_ints(E_pad);       // [E_pad] rank base of this CTA (running)
  int* s_off = base + E_pad;                     // [E+1]
  int* first = s_off + (E_pad + 4);              // [E] instance holding rank base[e]
  int* rbase = first + E_pad;                    // [R+1]
  int* i_cum = rbase + (R + 4);                  // inclusive cumulative quota
  int* i_dbase = i_cum + inst_cap;               // inst_base - cum_prev
  int* i_gbase = i_dbase + inst_cap;             // rank_base[rank] + i_dbase
  int* i_rank = i_gbase + inst_cap;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const int c = blockIdx.x;
  const long long cbegin = (long long)c * chunk_len;
  const int clen = (int)min((long long)chunk_len, (long long)S - cbegin);
  const bool has_gate = gate != nullptr;

  int ev[kRemapItems];
  GateT gv[kRemapItems];
  // loads of one round: warp w owns slots [w*span, (w+1)*span) of the round, step i covers
  // 32 consecutive slots (one coalesced 128-B line of ids)
  auto load_round = [&](int rbeg, int rlen, int items) {
    const int wbeg = rbeg + warp * items * 32;
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      const int off = wbeg + i * 32 + lane;
      const bool in = (i < items) && (off < rbeg + rlen);
      ev[i] = in ? __ldg(ids + cbegin + off) : -1;
      if (has_gate) gv[i] = in ? __ldg(gate + cbegin + off) : GateT(0);
    }
  };
  {
    const int rlen = min(kRemapRound, clen);
    load_round(0, rlen, (rlen + kRemapThreads - 1) / kRemapThreads);
  }

  // ---- stage the plan (coalesced, L2-resident) and this CTA's base ranks ---------------------
  for (int e = tid; e <= E; e += kRemapThreads) s_off[e] = g_inst_off[e];
  for (int r = tid; r <= R; r += kRemapThreads) rbase[r] = g_rank_base[r];
  for (int p = tid; p < inst_cap; p += kRemapThreads) {
    i_cum[p] = g_inst_cum[p];
    i_rank[p] = g_inst_rank[p];
    i_gbase[p] = g_inst_base[p];                 // raw inst_base for now
  }
  column_sums(table, c, E_pad, cnt, base);       // base[e] = sum of rows < c; syncs
  for (int p = tid; p < inst_cap; p += kRemapThreads) i_dbase[p] = (p > 0) ? i_cum[p - 1] : 0;
  __syncthreads();
  for (int e = tid; e < E; e += kRemapThreads) i_dbase[s_off[e]] = 0;   // first instance: cum_prev = 0
  __syncthreads();
  const int n_inst = s_off[E];
  for (int p = tid; p < n_inst; p += kRemapThreads) {
    const int d = i_gbase[p] - i_dbase[p];
    i_dbase[p] = d;
    i_gbase[p] = rbase[i_rank[p]] + d;
  }
  for (int e = tid; e < E; e += kRemapThreads) {                        // upper bound of base[e]
    const int lo = s_off[e];
    int a = 0, b = s_off[e + 1] - lo - 1;
    const int j = base[e];
    while (a < b) {
      const int mid = (a + b) >> 1;
      if (i_cum[lo + mid] > j) b = mid; else a = mid + 1;
    }
    first[e] = lo + a;
  }

  // ---- rounds of up to kRemapRound slots -----------------------------------------------------
  for (int rbeg = 0; rbeg < clen; rbeg += kRemapRound) {
    const int rlen = min(kRemapRound, clen - rbeg);
    const int items = (rlen + kRemapThreads - 1) / kRemapThreads;   // steps per warp, <= kRemapItems
    const int wbeg = rbeg + warp * items * 32;                      // offset inside the chunk
    if (rbeg > 0) {
      __syncthreads();                                              // previous round done with cnt
      load_round(rbeg, rlen, items);
    }
    for (int i = tid; i < kRemapWarps * E_pad; i += kRemapThreads) cnt[i] = 0;

    // peer masks: m = lanes with the same valid expert.  Packed into ev[i]:
    // e (bits 0..9) | rank among peers (10..14) | leader lane (15..19) | group size-1 (20..24); -1 invalid
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i < items) {
        const int e = ev[i];
        const bool valid = (unsigned)e < (unsigned)E;
        unsigned m = __ballot_sync(kFullMask, valid);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const bool bit = (e >> b) & 1;
          const unsigned bal = __ballot_sync(kFullMask, bit);
          m &= bit ? bal : ~bal;
        }
        const int r_in = __popc(m & lt_mask);
        const int leader = __ffs(m) - 1;
        ev[i] = valid ? (e | (r_in << 10) | (leader << 15) | ((__popc(m) - 1) << 20)) : -1;
      }
    }
    __syncthreads();                                                // cnt zeroed, plan staged

    // warp-private running counters: leaders add their group size in step order
    int* my = cnt + warp * E_pad;
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i < items) {
        const int pk = ev[i];
        int old = 0;
        if (pk >= 0 && ((pk >> 10) & 31) == 0) old = atomicAdd(&my[pk & 1023], ((pk >> 20) & 31) + 1);
        __syncwarp();                                               // orders step i before step i+1
        const int src = (pk >= 0) ? ((pk >> 15) & 31) : lane;
        old = __shfl_sync(kFullMask, old, src);
        if (pk >= 0) ev[i] = (pk & 1023) | ((old + ((pk >> 10) & 31)) << 10);   // e | rank in warp span
      }
    }
    __syncthreads();

    // cross-warp exclusive scan per expert column; cnt becomes the base of (warp, e)
    for (int e = tid; e < E; e += kRemapThreads) {
      int run = base[e];
#pragma unroll 8
      for (int w = 0; w < kRemapWarps; ++w) {
        const int x = cnt[w * E_pad + e];
        cnt[w * E_pad + e] = run;
        run += x;
      }
      base[e] = run;
    }
    __syncthreads();

#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      const int off = wbeg + i * 32 + lane;
      if (i < items && off < rbeg + rlen) {
        const long long s = cbegin + off;
        const int pk = ev[i];
        int rep = -1, rk = -1, of = -1;
        if (pk >= 0) {
          const int e = pk & 1023;
          const int j = my[e] + (pk >> 10);              // global stable rank among slots of e
          int p = first[e];
          const int last = s_off[e + 1] - 1;             // cum[last] = lambda_e > j when ws matches plan
          while (p < last && i_cum[p] <= j) ++p;
          rep = p - s_off[e];
          rk = i_rank[p];
          of = i_dbase[p] + j;
          if (has_gate) out_gate[i_gbase[p] + j] = gv[i];
        }
        out_replica[s] = rep;
        out_rank[s] = rk;
        out_offset[s] = of;
      }
    }
    if (rbeg + kRemapRound < clen) {                     // next round starts at base[e]: advance first
      __syncthreads();
      for (int e = tid; e < E; e += kRemapThreads) {
        int p = first[e];
        const int last = s_off[e + 1] - 1, j = base[e];
        while (p < last && i_cum[p] <= j) ++p;
        first[e] = p;
      }
    }
  }
}

template <typename GateT>
static int launch_remap_t(const Ctx* c, const int32_t* ids, const GateT* gate,
                          const uep_plan_out& p, int32_t* out_replica, int32_t* out_rank,
                          int32_t* out_offset, GateT* out_gate, void* ws, cudaStream_t s) {
  const uep_config& g = c->cfg;
  const int inst_cap = g.E + g.R * g.n_slot;
  const size_t smem = sizeof(int) * remap_smem_ints(c->E_pad, g.R, inst_cap);
  if (g.E > 256) {
    remap_kernel<GateT, 9><<<c->n_chunks, kRemapThreads, smem, s>>>(
        ids, gate, c->S, g.E, c->E_pad, g.R, inst_cap, c->chunk_len, ws_table(ws), p.inst_off,
        p.inst_rank, p.inst_cum, p.inst_base, p.rank_base, out_replica, out_rank, out_offset, out_gate);
  } else {
    remap_kernel<GateT, 8><<<c->n_chunks, kRemapThreads, smem, s>>>(
        ids, gate, c->S, g.E, c->E_pad, g.R, inst_cap, c->chunk_len, ws_table(ws), p.inst_off,
        p.inst_rank, p.inst_cum, p.inst_base, p.rank_base, out_replica, out_rank, out_offset, out_gate);
  }
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

int init_remap_kernels() {
  const int bytes = (int)(sizeof(int) * remap_smem_ints(UEP_MAX_E, UEP_MAX_R, kMaxInst));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint32_t, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint32_t, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint16_t, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint16_t, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  return UEP_OK;
}

int launch_remap(const Ctx* c, const int32_t* ids, const void* gate, const uep_plan_out& p,
                 int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                 void* ws, cudaStream_t s) {
  if (c->S == 0) return UEP_OK;
  if (c->cfg.gate_dtype == UEP_GATE_BF16 && gate)
    return launch_remap_t<uint16_t>(c, ids, static_cast<const uint16_t*>(gate), p, out_replica,
                                    out_rank, out_offset, static_cast<uint16_t*>(out_gate), ws, s);
  return launch_remap_t<uint32_t>(c, ids, static_cast<const uint32_t*>(gate), p, out_replica,
                                  out_rank, out_offset, static_cast<uint32_t*>(out_gate), ws, s);
}

}  // namespace uep
