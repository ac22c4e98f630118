// remap.cu — uep_remap: token assignment (§5.2 "Token Assignment").
//
// For slot s with expert e: j = global stable rank of s among the slots of e; instance
// i = first whose cumulative quota exceeds j (upper-bound lookup); destination
// (rank, offset) inside that rank's receive buffer; gate copied bit-exact (moved as raw
// 16/32-bit integers, S17).
//
// HBM-bound by its bytes (4 B id + g B gate read, 12 B + g B written per slot), but on a
// 50 MB problem the limiter is the INSTRUCTION count of the stable ranking (integer pipes
// issue one warp instruction per two cycles), so the kernel is built to rank a slot in as
// few instructions as possible:
//   * one CTA per chunk, every warp owns a contiguous span and loads its ids and gates up
//     front (coalesced 128 B per warp-load, unpredicated when the round is full);
//   * ranking inside a warp uses a warp-private shared-memory row of {peer mask, count} cells:
//     lanes OR their lane bit into the cell of their expert, read {mask, count} back with one
//     64-bit load, and the lowest peer stores {0, count + popc(mask)}.  Rank = count +
//     popc(mask & lower lanes): stable by construction, no order-dependent atomic result is
//     ever used (the OR is commutative);
//   * one cross-warp scan per expert column turns the counts into CTA-wide bases; the CTA's own
//     base comes from summing the chunk-table rows below it (independent int4 L2 loads, in
//     flight together with the id loads);
//   * lookup: per CTA and expert one 16-B record describes the instance holding the CTA's first
//     slot of that expert; a slot only walks further when it crosses a quota edge;
//   * gates are staged in shared memory in (expert, rank) order and written as contiguous runs
//     (a scatter of 4-B stores costs one L2 request per lane).
#include "uep_internal.cuh"

namespace uep {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr size_t kMaxSmem = 227 * 1024;

// dynamic shared memory layout (ints):
//   wrow[kRemapWarps][E_pad] (int2) | rec[E_pad] (int4) | base[E_pad] | base0[E_pad] | elb[E_pad]
//   | s_off[E_pad+4] | rbase[(R+7)&~3] | i_cum | i_dbase | i_gbase | i_rank (inst_cap each) | wtot[32]
//   | scratch: part[kColPartInts] during staging, then (STAGE) the gate staging buffer
__host__ __device__ inline size_t remap_fixed_ints(int E_pad, int R, int inst_cap) {
  return 2 * (size_t)kRemapWarps * E_pad + 4 * (size_t)E_pad + 3 * (size_t)E_pad + (E_pad + 4) +
         ((R + 7) & ~3) + 4 * (size_t)((inst_cap + 3) & ~3) + 32;
}
__host__ __device__ inline size_t remap_smem_bytes(int E_pad, int R, int inst_cap, bool stage,
                                                   int gate_bytes) {
  size_t scratch = sizeof(int) * (size_t)kColPartInts;
  const size_t sg = (size_t)kRemapRound * gate_bytes;
  if (stage && sg > scratch) scratch = sg;
  return sizeof(int) * remap_fixed_ints(E_pad, R, inst_cap) + scratch;
}

template <typename GateT, bool STAGE>
__global__ void __launch_bounds__(kRemapThreads, 1)
remap_kernel(const int32_t* __restrict__ ids, const GateT* __restrict__ gate, int S, int E,
             int E_pad, int R, int inst_cap, int chunk_len, const int32_t* __restrict__ table,
             const int32_t* __restrict__ g_inst_off, const int32_t* __restrict__ g_inst_rank,
             const int32_t* __restrict__ g_inst_cum, const int32_t* __restrict__ g_inst_base,
             const int32_t* __restrict__ g_rank_base, int32_t* __restrict__ out_replica,
             int32_t* __restrict__ out_rank, int32_t* __restrict__ out_offset,
             GateT* __restrict__ out_gate) {
  extern __shared__ __align__(16) int smem[];
  int2* wrow = reinterpret_cast<int2*>(smem);                       // [warps][E_pad] {mask, count}
  int4* rec = reinterpret_cast<int4*>(wrow + kRemapWarps * E_pad);  // [E_pad] fast-path record
  int* base = reinterpret_cast<int*>(rec + E_pad);                  // [E_pad] running rank base of the CTA
  int* base0 = base + E_pad;                     // [E_pad] base at the start of the round
  int* elb = base0 + E_pad;                      // [E_pad] staging position of rank j is elb[e] + j
  int* s_off = elb + E_pad;                      // [E+1]
  int* rbase = s_off + (E_pad + 4);              // [R+1]
  const int icap = (inst_cap + 3) & ~3;
  int* i_cum = rbase + ((R + 7) & ~3);           // inclusive cumulative quota
  int* i_dbase = i_cum + icap;                   // inst_base - cum_prev
  int* i_gbase = i_dbase + icap;                 // rank_base[rank] + i_dbase
  int* i_rank = i_gbase + icap;
  int* wtot = i_rank + icap;                     // [32]
  int* part = wtot + 32;                         // column-sum partials (staging only)
  GateT* sg = reinterpret_cast<GateT*>(part);    // gate staging buffer (after staging)

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned lane_bit = 1u << lane, lt_mask = lane_bit - 1u;
  const int c = blockIdx.x;
  const long long cbegin = (long long)c * chunk_len;
  const int clen = (int)min((long long)chunk_len, (long long)S - cbegin);
  const bool has_gate = gate != nullptr;
  ids += cbegin; out_replica += cbegin; out_rank += cbegin; out_offset += cbegin;
  if (has_gate) gate += cbegin;

  int ev[kRemapItems];
  GateT gv[kRemapItems];
  // loads of one round: warp w owns slots [w*span, (w+1)*span) of the round, step i covers
  // 32 consecutive slots (one coalesced 128-B line of ids)
  auto load_round = [&](int wbeg, int rend, int items, bool full) {
    const int32_t* ip = ids + wbeg + lane;
    const GateT* gp = gate + wbeg + lane;
    if (full) {
#pragma unroll
      for (int i = 0; i < kRemapItems; ++i) {
        if (i < items) {
          ev[i] = __ldg(ip + i * 32);
          if (has_gate) gv[i] = __ldg(gp + i * 32);
        }
      }
    } else {
      const int room = rend - wbeg - lane;                        // slot i*32 is in range iff i*32 < room
#pragma unroll
      for (int i = 0; i < kRemapItems; ++i) {
        const bool in = (i < items) && (i * 32 < room);
        ev[i] = in ? __ldg(ip + i * 32) : -1;
        if (has_gate) gv[i] = in ? __ldg(gp + i * 32) : GateT(0);
      }
    }
  };
  {
    const int rlen = min(kRemapRound, clen);
    const int items = (rlen + kRemapThreads - 1) / kRemapThreads;
    load_round(warp * items * 32, rlen, items, rlen == items * kRemapThreads);
  }

  // ---- this CTA's base ranks: column sums of the table rows below its own (loads in flight) ----
  const int CG = E_pad >> 2;
  const int NRG = min(32, kRemapThreads / CG);
  {
    const int cg = tid % CG, rg = tid / CG;
    if (rg < NRG) {
      int4 acc = make_int4(0, 0, 0, 0);
      const int4* col = reinterpret_cast<const int4*>(table) + cg;
#pragma unroll 10
      for (int r = rg; r < c; r += NRG) {
        const int4 v = __ldcg(col + (size_t)r * CG);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
      }
      reinterpret_cast<int4*>(part)[rg * CG + cg] = acc;
    }
  }
  // ---- stage the plan (coalesced, L2-resident) ---------------------------------------------------
  for (int e = tid; e <= E; e += kRemapThreads) s_off[e] = g_inst_off[e];
  for (int r = tid; r <= R; r += kRemapThreads) rbase[r] = g_rank_base[r];
  for (int p = tid; p < inst_cap; p += kRemapThreads) {
    const int cum = g_inst_cum[p];
    i_cum[p] = cum;
    i_rank[p] = g_inst_rank[p];
    i_gbase[p] = g_inst_base[p];                 // raw inst_base for now
    if (p + 1 < inst_cap) i_dbase[p + 1] = cum;  // cum_prev of the next entry
    if (p == 0) i_dbase[0] = 0;
  }
  {
    int4* z = reinterpret_cast<int4*>(wrow);
    for (int i = tid; i < kRemapWarps * E_pad / 2; i += kRemapThreads) z[i] = make_int4(0, 0, 0, 0);
  }
  __syncthreads();
  for (int e = tid; e < E_pad; e += kRemapThreads) {
    int sum = 0;
    for (int g = 0; g < NRG; ++g) sum += part[g * E_pad + e];
    base[e] = sum;
    if (e < E) i_dbase[s_off[e]] = 0;            // first instance of an expert: cum_prev = 0
  }
  __syncthreads();
  const int n_inst = s_off[E];
  for (int p = tid; p < n_inst; p += kRemapThreads) {
    const int d = i_gbase[p] - i_dbase[p];
    i_dbase[p] = d;
    i_gbase[p] = rbase[i_rank[p]] + d;
  }
  __syncthreads();
  // rec[e] = {cum, dbase, gbase, rep<<16|rank} of the instance holding rank base[e]
  auto make_rec = [&](int e, int pstart) {
    const int lo = s_off[e], last = s_off[e + 1] - 1, j = base[e];
    int p = pstart < lo ? lo : pstart;
    while (p < last && i_cum[p] <= j) ++p;
    rec[e] = make_int4(i_cum[p], i_dbase[p], i_gbase[p], ((p - lo) << 16) | i_rank[p]);
  };
  for (int e = tid; e < E; e += kRemapThreads) make_rec(e, 0);

  // ---- rounds of up to kRemapRound slots -----------------------------------------------------
  for (int rbeg = 0; rbeg < clen; rbeg += kRemapRound) {
    const int rlen = min(kRemapRound, clen - rbeg);
    const int items = (rlen + kRemapThreads - 1) / kRemapThreads;   // steps per warp, <= kRemapItems
    const int wbeg = rbeg + warp * items * 32;                      // offset inside the chunk
    const bool full = (rlen == items * kRemapThreads);
    if (rbeg > 0) {
      __syncthreads();                                              // previous round done with wrow, rec, sg
      load_round(wbeg, rbeg + rlen, items, full);
      int4* z = reinterpret_cast<int4*>(wrow);
      for (int i = tid; i < kRemapWarps * E_pad / 2; i += kRemapThreads) z[i] = make_int4(0, 0, 0, 0);
      for (int e = tid; e < E; e += kRemapThreads) make_rec(e, s_off[e] + (rec[e].w >> 16));
    }
    __syncthreads();                                                // rows zeroed, plan staged, rec ready

    // stable rank inside the warp span: steps in order, lanes in order
    int2* wr = wrow + warp * E_pad;
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i < items) {
        const int e = ev[i];
        const bool valid = (unsigned)e < (unsigned)E;
        int2* cell = wr + (valid ? e : 0);
        if (valid) atomicOr(reinterpret_cast<unsigned*>(&cell->x), lane_bit);
        __syncwarp();
        const int2 mc = *cell;                                      // {peer mask, count so far}
        __syncwarp();
        const unsigned m = (unsigned)mc.x;
        if (valid && (m & lt_mask) == 0u) *cell = make_int2(0, mc.y + __popc(m));   // lowest peer
        __syncwarp();                                               // cell cleared before the next step
        ev[i] = valid ? (e | ((mc.y + __popc(m & lt_mask)) << 10)) : -1;   // e | rank in warp span
      }
    }
    __syncthreads();

    // cross-warp exclusive scan per expert column; the count field becomes the base of (warp, e)
    {
      int n = 0, old = 0;
      if (tid < E) {
        int run = base[tid];
        old = run;
#pragma unroll 8
        for (int w = 0; w < kRemapWarps; ++w) {
          const int x = wrow[w * E_pad + tid].y;
          wrow[w * E_pad + tid].y = run;
          run += x;
        }
        base[tid] = run;
        base0[tid] = old;
        n = run - old;
      }
      if (STAGE && has_gate) {                                      // staging offsets: scan of n over e
        int inc = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int y = __shfl_up_sync(kFullMask, inc, o);
          if (lane >= o) inc += y;
        }
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        int pre = 0;
        for (int w = 0; w < warp; ++w) pre += wtot[w];
        if (tid < E) elb[tid] = pre + inc - n - old;
      }
    }
    __syncthreads();

    int32_t* o_rep = out_replica + wbeg + lane;
    int32_t* o_rnk = out_rank + wbeg + lane;
    int32_t* o_off = out_offset + wbeg + lane;
    const int room = full ? 0x7fffffff : rbeg + rlen - wbeg - lane;
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i < items && i * 32 < room) {
        const int pk = ev[i];
        int rep = -1, rk = -1, of = -1;
        if (pk >= 0) {
          const int e = pk & 1023;
          const int j = wr[e].y + (pk >> 10);            // global stable rank among slots of e
          const int4 rc = rec[e];
          int db = rc.y, gb = rc.z, rr = rc.w;
          if (j >= rc.x) {                               // past the first instance of this CTA's window
            int p = s_off[e] + (rr >> 16) + 1;
            const int last = s_off[e + 1] - 1;           // cum[last] = lambda_e > j when ws matches plan
            while (p < last && i_cum[p] <= j) ++p;
            db = i_dbase[p]; gb = i_gbase[p]; rr = ((p - s_off[e]) << 16) | i_rank[p];
          }
          rep = rr >> 16;
          rk = rr & 0xffff;
          of = db + j;
          if (has_gate) {
            if (STAGE) sg[elb[e] + j] = gv[i];
            else out_gate[gb + j] = gv[i];
          }
        }
        o_rep[i * 32] = rep;
        o_rnk[i * 32] = rk;
        o_off[i * 32] = of;
      }
    }

    if (STAGE && has_gate) {                             // write the staged gates as contiguous runs
      __syncthreads();
      for (int e = warp; e < E; e += kRemapWarps) {
        const int j1 = base[e], off = elb[e];
        int p = s_off[e] + (rec[e].w >> 16);
        const int last = s_off[e + 1] - 1;
        for (int j = base0[e] + lane; j < j1; j += 32) {
          while (p < last && i_cum[p] <= j) ++p;
          out_gate[i_gbase[p] + j] = sg[off + j];
        }
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
  const bool stage = gate && remap_smem_bytes(c->E_pad, g.R, inst_cap, true, sizeof(GateT)) <= kMaxSmem;
  const size_t smem = remap_smem_bytes(c->E_pad, g.R, inst_cap, stage, sizeof(GateT));
  auto k = stage ? remap_kernel<GateT, true> : remap_kernel<GateT, false>;
  k<<<c->n_chunks, kRemapThreads, smem, s>>>(
      ids, gate, c->S, g.E, c->E_pad, g.R, inst_cap, c->chunk_len, ws_table(ws), p.inst_off,
      p.inst_rank, p.inst_cum, p.inst_base, p.rank_base, out_replica, out_rank, out_offset, out_gate);
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

int init_remap_kernels() {
  const int bytes = (int)kMaxSmem;
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint32_t, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint32_t, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint16_t, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(remap_kernel<uint16_t, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
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
