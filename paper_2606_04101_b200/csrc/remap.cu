// remap.cu — uep_remap: token assignment (§5.2 "Token Assignment").
//
// For slot s with expert e: j = global stable rank of s among the slots of e; instance
// i = first whose cumulative quota exceeds j (upper-bound lookup); destination
// (rank, offset) inside that rank's receive buffer; gate copied bit-exact (moved as raw
// 16/32-bit integers, S17).
//
// HBM-bound: 4 B id + g B gate read, 12 B + g B written per slot (24 B/slot for fp32 gates).
// It is a stable 512-bin multi-split: one CTA per chunk (the chunk prefix table comes from
// uep_histogram), every warp owns a contiguous span of the chunk, loads all its ids and gates
// up front (coalesced 128 B per warp-load), ranks them with match.any + a warp-private
// shared-memory counter row, then one cross-warp scan per expert column gives the CTA-wide
// stable rank.  No atomics: the result is the stable order by construction.
#include "uep_internal.cuh"

namespace uep {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr int kMaxInst = UEP_MAX_E + UEP_MAX_R * UEP_MAX_NSLOT;   // 1536 CSR entries at most

// dynamic shared memory layout (ints): cnt[kRemapWarps][E_pad] | base[E_pad] | inst_off[E_pad+1]
// | i_cum[n_inst] | i_dbase[n_inst] | i_gbase[n_inst] | i_rank[n_inst]
__host__ __device__ inline size_t remap_smem_ints(int E_pad, int inst_cap) {
  return (size_t)kRemapWarps * E_pad + E_pad + (E_pad + 1) + 4 * (size_t)inst_cap;
}

template <typename GateT>
__global__ void __launch_bounds__(kRemapThreads, 1)
remap_kernel(const int32_t* __restrict__ ids, const GateT* __restrict__ gate, int S, int E,
             int E_pad, int P, int inst_cap, int chunk_len, const int32_t* __restrict__ table,
             const int32_t* __restrict__ g_inst_off, const int32_t* __restrict__ g_inst_rank,
             const int32_t* __restrict__ g_inst_phys, const int32_t* __restrict__ g_inst_cum,
             const int32_t* __restrict__ g_phys_base, const int32_t* __restrict__ g_rank_base,
             int32_t* __restrict__ out_replica, int32_t* __restrict__ out_rank,
             int32_t* __restrict__ out_offset, GateT* __restrict__ out_gate) {
  extern __shared__ __align__(16) int smem[];
  int* cnt = smem;                               // [warps][E_pad]
  int* base = cnt + kRemapWarps * E_pad;         // [E_pad] running rank base of this CTA
  int* s_off = base + E_pad;                     // [E_pad+1]
  int* i_cum = s_off + (E_pad + 1);              // inclusive cumulative quota
  int* i_dbase = i_cum + inst_cap;               // phys_base[rank][phys] - cum_prev
  int* i_gbase = i_dbase + inst_cap;             // rank_base[rank] + i_dbase
  int* i_rank = i_gbase + inst_cap;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c = blockIdx.x;
  const long long cbegin = (long long)c * chunk_len;
  const int clen = (int)min((long long)chunk_len, (long long)S - cbegin);
  const bool has_gate = gate != nullptr;

  // ---- stage the plan (small, L2-resident) -------------------------------------------------
  for (int e = tid; e <= E; e += kRemapThreads) s_off[e] = g_inst_off[e];
  for (int e = tid; e < E_pad; e += kRemapThreads)
    base[e] = (e < E) ? __ldcg(table + (size_t)c * E_pad + e) : 0;
  __syncthreads();
  for (int e = tid; e < E; e += kRemapThreads) {
    const int lo = s_off[e], hi = s_off[e + 1];
    int prev = 0;
    for (int p = lo; p < hi; ++p) {
      const int r = g_inst_rank[p], ph = g_inst_phys[p], cum = g_inst_cum[p];
      const int db = g_phys_base[r * P + ph] - prev;
      i_cum[p] = cum;
      i_dbase[p] = db;
      i_gbase[p] = g_rank_base[r] + db;
      i_rank[p] = r;
      prev = cum;
    }
  }

  // ---- rounds of up to kRemapRound slots -----------------------------------------------------
  for (int rbeg = 0; rbeg < clen; rbeg += kRemapRound) {
    const int rlen = min(kRemapRound, clen - rbeg);
    const int items = (rlen + kRemapThreads - 1) / kRemapThreads;   // steps per warp, <= kRemapItems
    const int span = items * 32;                                    // slots per warp this round
    const int wbeg = rbeg + warp * span;                            // offset inside the chunk
    for (int i = tid; i < kRemapWarps * E_pad; i += kRemapThreads) cnt[i] = 0;

    int ev[kRemapItems];
    GateT gv[kRemapItems];
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      const int off = wbeg + i * 32 + lane;
      const bool in = (i < items) && (off < rbeg + rlen);
      ev[i] = in ? __ldg(ids + cbegin + off) : -1;
      if (has_gate && in) gv[i] = __ldg(gate + cbegin + off);
    }
    __syncthreads();                                                // cnt zeroed (and plan staged)

    // stable rank inside the warp span: lower steps first, lower lanes first
    int* my = cnt + warp * E_pad;
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i < items) {
        const int e = ev[i];
        const bool valid = (unsigned)e < (unsigned)E;
        const unsigned m = __match_any_sync(kFullMask, valid ? e : -1);
        const unsigned lower = m & ((1u << lane) - 1u);
        const int cur = valid ? my[e] : 0;
        const int r = cur + __popc(lower);
        __syncwarp();                                        // every peer has read the counter
        if (valid && lower == 0u) my[e] = cur + __popc(m);   // group leader (lowest lane)
        __syncwarp();
        ev[i] = valid ? (e | (r << 16)) : -1;
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
          const int e = pk & 0xffff, r = pk >> 16;
          const int j = my[e] + r;                       // global stable rank among slots of e
          const int lo = s_off[e], n = s_off[e + 1] - lo;
          int a = 0;
          if (n > 1) {                                   // upper bound: first cum > j
            int b = n - 1;                               // cum[last] = lambda_e > j always
            while (a < b) {
              const int mid = (a + b) >> 1;
              if (i_cum[lo + mid] > j) b = mid; else a = mid + 1;
            }
          }
          rep = a;
          rk = i_rank[lo + a];
          of = i_dbase[lo + a] + j;
          if (has_gate) out_gate[i_gbase[lo + a] + j] = gv[i];
        }
        out_replica[s] = rep;
        out_rank[s] = rk;
        out_offset[s] = of;
      }
    }
    __syncthreads();                                     // cnt is re-zeroed by the next round
  }
}

int init_remap_kernels() {
  const int bytes = (int)(sizeof(int) * remap_smem_ints(UEP_MAX_E, kMaxInst));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint16_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  return UEP_OK;
}

int launch_remap(const Ctx* c, const int32_t* ids, const void* gate, const uep_plan_out& p,
                 int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                 void* ws, cudaStream_t s) {
  if (c->S == 0) return UEP_OK;
  const uep_config& g = c->cfg;
  const int inst_cap = g.E + g.R * g.n_slot;
  const size_t smem = sizeof(int) * remap_smem_ints(c->E_pad, inst_cap);
  if (g.gate_dtype == UEP_GATE_BF16 && gate) {
    remap_kernel<uint16_t><<<c->n_chunks, kRemapThreads, smem, s>>>(
        ids, static_cast<const uint16_t*>(gate), c->S, g.E, c->E_pad, c->P, inst_cap,
        c->chunk_len, ws_table(ws), p.inst_off, p.inst_rank, p.inst_phys, p.inst_cum, p.phys_base,
        p.rank_base, out_replica, out_rank, out_offset, static_cast<uint16_t*>(out_gate));
  } else {
    remap_kernel<uint32_t><<<c->n_chunks, kRemapThreads, smem, s>>>(
        ids, static_cast<const uint32_t*>(gate), c->S, g.E, c->E_pad, c->P, inst_cap, c->chunk_len,
        ws_table(ws), p.inst_off, p.inst_rank, p.inst_phys, p.inst_cum, p.phys_base, p.rank_base,
        out_replica, out_rank, out_offset, static_cast<uint32_t*>(out_gate));
  }
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

}  // namespace uep
