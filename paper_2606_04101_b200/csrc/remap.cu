// remap.cu — uep_remap: token assignment (§5.2 "Token Assignment").
//
// For slot s with expert e: j = global stable rank of s among the slots of e; instance
// i = first whose cumulative quota exceeds j (upper-bound lookup); destination
// (rank, offset) inside that rank's receive buffer; gate copied bit-exact (moved as raw
// 16/32-bit integers, S17).
//
// Two kernels, split at the only data dependence on the plan:
//   rank_kernel   (plan-INDEPENDENT) stable rank of every slot among the slots of the same
//                 expert inside its chunk, packed with the expert id into one int32 per slot in
//                 the workspace.  uep_balance runs it on a side stream concurrently with
//                 uep_histogram and uep_plan, so it is off the critical path gate -> dispatch.
//   lookup_kernel (plan-DEPENDENT) global rank = chunk base (the chunk's row of the exclusive
//                 prefix over chunks, left by prefix_kernel) + rank in chunk; cumulative-quota
//                 lookup; writes (replica, rank, offset) and the gates in dispatch order.  Under
//                 programmatic dependent launch everything before its griddepcontrol.wait (the
//                 loads of packed ranks and gates) overlaps the planner.
//
// The source-aware variant (uep_remap_local, SolveReroute of Alg. 1 lines 26-36) reuses the same
// kernels on chunks that never straddle a source rank's block of tokens, with reroute_kernel
// (below) in between to decompose the quotas per source rank.
//
// rank_kernel: one CTA per chunk (<= 8192 slots, register-resident, two CTAs per SM), every warp owns a
// contiguous span and loads its ids up front (coalesced).  Ranking inside a warp uses a
// warp-private shared-memory row of {peer mask, count} cells: lanes OR their lane bit into the
// cell of their expert, read {mask, count} back with one 64-bit load, and the lowest peer stores
// {0, count + popc(mask)}.  Rank = count + popc(mask & lower lanes): stable by construction, no
// order-dependent atomic result is ever used (the OR is commutative).  (Measured alternative:
// peers found with match.any.sync instead of the OR + read-back: 19.7 us for rank + prefix at
// the DeepSeek-V3 shape against 11.8 us — MATCH.ANY is the slower instruction.)  One cross-warp scan per
// expert column turns the counts into chunk-wide bases and gives the chunk's row of a count
// table, which prefix_kernel (a thread per row, a CTA per four columns) scans over chunks.
//
// lookup_kernel: per CTA and expert one 16-B record describes the instance holding the CTA's
// first slot of that expert; a slot only walks further when it crosses a quota edge.  Gates are
// staged in shared memory in (expert, rank) order together with their destination index and
// written out as contiguous runs (a scatter of 4-B stores costs one L2 request per lane).
// (Measured alternative: four consecutive slots per thread with 16-B loads and stores — fewer
// instructions, but 15.2 us against 14.5 us: at 7168 slots per CTA half of the warps get a
// fourth group and the others wait for them.)
#include "uep_internal.cuh"

namespace uep {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr int kEMask = (1 << kPackedEBits) - 1;

// ------------------------------------------------------------------------------------------------
// rank_kernel.  Two ways to the same packed words (expert | stable rank inside the chunk << 9):
//
// FAST (W > 0), for routing as top-k produces it — a token names an expert at most once.  Then the
// slots of expert e in the chunk are one per token, in token order, and the rank of slot (t, e) is
// the number of tokens before t that name e: a bitmap per expert over the chunk's tokens
// (B[e][W] words), one shared-memory atomicOr per slot (commutative: no order-dependent atomic
// anywhere), an exclusive prefix of the words' popcounts per expert (P[e][W], 16 bit), and
// rank = P[e][w] + popc(B[e][w] & bits below t).  Every slot of a thread is independent of the
// others (no warp-synchronous steps).  An atomicOr that finds its bit already set has met a token
// that names an expert twice: the CTA then falls back to the general way below.
// dynamic shared memory: B[E_pad][W] (int32) | P[E_pad][W] (uint16)
//
// GENERAL (any ids; W == 0 when the bitmaps do not fit or k is 1): every warp owns a row of cells
// {peer mask, count} per expert and ranks its span in steps of 32 slots (lanes in order): atomicOr
// of the lane's bit, read, the lowest peer adds the popcount and clears the mask.
// dynamic shared memory: wrow[kRemapWarps][E_pad] (int2 {mask, count})
// ------------------------------------------------------------------------------------------------
constexpr size_t kRankFastSmem = 96 * 1024;        // two CTAs per SM beside the other kernels of the chain

// words per expert row of the token bitmaps for chunks of chunk_len slots, 0 = general way only
inline int rank_fast_words(int chunk_len, int k, int E_pad) {
  if (k < 2 || k > 64) return 0;                   // (k = 1: one slot per token, nothing to gain; the division by
  const int toks = chunk_len / k + 2;              //  multiplication below is exact for slot * k < 2^32)
  const int W = ((toks + 31) / 32) | 1;            // odd pitch: rows of different experts start in different banks
  return (size_t)E_pad * W * 6 <= kRankFastSmem ? W : 0;
}
inline size_t rank_smem_bytes(int E_pad, int W) {
  const size_t general = sizeof(int2) * (size_t)kRemapWarps * E_pad, fast = (size_t)E_pad * W * 6 + 16;
  return general > fast ? general : fast;
}

// BITMAPS = false is the general way alone, with the code the compiler makes for it alone (uep_balance
// launches that one: 42 registers, so that a CTA fits beside the planner's 512 x 80 on one SM; inside
// the BITMAPS = true kernel the general loop comes out at 39 instructions per step instead of 30).
template <bool BITMAPS>
__global__ void __launch_bounds__(kRemapThreads, 2)
rank_kernel(const int32_t* __restrict__ ids, int S, int E, int E_pad, int chunk_len, int cpg,
            int group_len, int32_t* __restrict__ packed, int32_t* __restrict__ prefix,
            int32_t* __restrict__ counts, int chunk0, int W, unsigned k_magic, int early_trigger) {
  extern __shared__ __align__(16) int smem[];
  int2* wrow = reinterpret_cast<int2*>(smem);
  // prefix_kernel may be scheduled (it waits for this grid).  Not when the kernel behind this one is
  // the lookup itself (uep_shard_count: under stream capture the lookup's edge from this kernel is
  // programmatic, and its prologue reads what this kernel writes)
  if (early_trigger) pdl_trigger();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned lane_bit = 1u << lane, lt_mask = lane_bit - 1u;
  const int cb = (int)blockIdx.x + chunk0;       // chunk0 > 0: a token shard's CTAs (uep_shard_count)
  // chunk c = sub-chunk c % cpg of group c / cpg (a group = one source rank's slots in the
  // source-aware remap; the whole input, cpg = number of chunks, otherwise)
  const int sub = cb % cpg;
  const long long cbegin = (long long)(cb / cpg) * group_len + (long long)sub * chunk_len;
  const int clen = (int)min(min((long long)chunk_len, (long long)group_len - (long long)sub * chunk_len),
                            (long long)S - cbegin);                            // <= kMaxChunk
  const int items = (clen + kRemapThreads - 1) / kRemapThreads;                // steps per warp
  const bool full = (clen == items * kRemapThreads);
  const int wbeg = warp * items * 32;
  const int room = full ? 0x7fffffff : clen - wbeg - lane;   // step i in range iff i*32 < room
  ids += cbegin + wbeg + lane;
  packed += cbegin + wbeg + lane;

  int ev[kRemapItems];
#pragma unroll
  for (int i = 0; i < kRemapItems; ++i)
    ev[i] = (i < items && i * 32 < room) ? __ldg(ids + i * 32) : -1;

  if (BITMAPS && W > 0) {
    int* B = smem;
    unsigned short* P = reinterpret_cast<unsigned short*>(B + E_pad * W);
    {
      int4* z = reinterpret_cast<int4*>(B);                            // E_pad % 4 == 0
      for (int i = tid; i < E_pad * W / 4; i += kRemapThreads) z[i] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    // token of slot g (global index) = g / k = umulhi(g, ceil(2^32 / k)), exact for g * k < 2^32
    const unsigned tok0 = __umulhi((unsigned)cbegin, k_magic);
    const unsigned g0 = (unsigned)cbegin + (unsigned)(wbeg + lane);
    unsigned dup = 0;
    const unsigned B_s = smem_u32(B);
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) {
      if (i >= items) break;                                            // (CTA-uniform)
      const unsigned e = (unsigned)ev[i];
      const bool valid = e < (unsigned)E;                               // (a slot beyond the chunk holds -1)
      const unsigned lt = __umulhi(g0 + 32u * i, k_magic) - tok0;       // token inside the chunk
      const unsigned bit = 1u << (lt & 31u);
      unsigned old = 0;                                                 // (a predicated atomic, no branch per slot)
      asm volatile("{ .reg .pred p; setp.ne.u32 p, %4, 0; @p atom.shared.or.b32 %0, [%1], %2; @!p mov.u32 %0, %3; }"
                   : "=r"(old) : "r"(B_s + 4u * (e * (unsigned)W + (lt >> 5))), "r"(bit), "r"(0u), "r"((unsigned)valid) : "memory");
      dup |= old & bit;
      ev[i] = valid ? (int)(e | (lt << kPackedEBits)) : -1;
    }
    if (!__syncthreads_or(dup != 0u)) {
      // per expert: exclusive prefix of the words' popcounts; the total is the chunk's count of e
      for (int e = tid; e < E_pad; e += kRemapThreads) {
        int run = 0;
#pragma unroll 4
        for (int w = 0; w < W; ++w) {
          P[e * W + w] = (unsigned short)run;
          run += __popc((unsigned)B[e * W + w]);
        }
        prefix[(size_t)(cb + 1) * E_pad + e] = run;     // (rows of e >= E are all zero)
        if (counts) counts[(size_t)cb * E_pad + e] = run;
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < kRemapItems; ++i) {
        if (i >= items) break;                                          // (CTA-uniform)
        const int pk = ev[i];
        const unsigned up = (unsigned)max(pk, 0);                       // (-1: cell 0, result unused)
        const unsigned e = up & (unsigned)kEMask, lt = up >> kPackedEBits;
        const unsigned idx = e * (unsigned)W + (lt >> 5);
        const int r = (int)P[idx] + __popc((unsigned)B[idx] & ((1u << (lt & 31u)) - 1u));
        if (i * 32 < room) packed[i * 32] = pk >= 0 ? (int)(e | ((unsigned)r << kPackedEBits)) : -1;
      }
      return;
    }
    // a token names an expert twice: redo the chunk the general way (the barrier above ordered every
    // atomicOr before the cells below are cleared)
#pragma unroll
    for (int i = 0; i < kRemapItems; ++i) ev[i] = ev[i] < 0 ? -1 : (ev[i] & kEMask);
  }

  {
    int4* z = reinterpret_cast<int4*>(wrow);
    for (int i = tid; i < kRemapWarps * E_pad / 2; i += kRemapThreads) z[i] = make_int4(0, 0, 0, 0);
  }
  __syncthreads();

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
      const int2 mc = *cell;                                        // {peer mask, count so far}
      __syncwarp();
      const unsigned m = (unsigned)mc.x;
      if (valid && (m & lt_mask) == 0u) *cell = make_int2(0, mc.y + __popc(m));   // lowest peer
      __syncwarp();                                                 // cell cleared before the next step
      ev[i] = valid ? (e | ((mc.y + __popc(m & lt_mask)) << kPackedEBits)) : -1;
    }
  }
  __syncthreads();

  // cross-warp exclusive scan per expert column; the count field becomes the base of (warp, e);
  // the column total is this chunk's row of the count table (row c+1: row 0 stays zero, so that
  // the in-place inclusive scan over rows below leaves the EXCLUSIVE prefix in row c)
  for (int e = tid; e < E_pad; e += kRemapThreads) {
    int run = 0;
    if (e < E) {
#pragma unroll 8
      for (int w = 0; w < kRemapWarps; ++w) {
        const int x = wrow[w * E_pad + e].y;
        wrow[w * E_pad + e].y = run;
        run += x;
      }
    }
    prefix[(size_t)(cb + 1) * E_pad + e] = run;
    if (counts) counts[(size_t)cb * E_pad + e] = run;     // row c of `counts` is never rewritten: the lookup reads it before prefix_kernel is done
  }
  __syncthreads();

#pragma unroll
  for (int i = 0; i < kRemapItems; ++i) {
    if (i < items && i * 32 < room) {
      const int pk = ev[i];
      packed[i * 32] = (pk >= 0) ? pk + (wr[pk & kEMask].y << kPackedEBits) : -1;
    }
  }
}

// prefix_kernel: rows 1..n_rows of the count table hold per-chunk counts (row 0 is zero);
// inclusive scan over rows, in place, turns row c into the EXCLUSIVE prefix of chunk c and row
// n_rows into the totals.  One CTA per int4 column group, one thread per row (blocks of 1024
// rows with a carry): one L2 round trip per block instead of a serial walk.
__global__ void __launch_bounds__(1024, 1)
prefix_kernel(int32_t* __restrict__ prefix, int n_rows, int CG) {
  __shared__ int4 wsum[32];
  // launched programmatically dependent on rank_kernel: wait for it, and only then let the kernel
  // behind this one (the lookup) start: its prologue reads what rank_kernel wrote, and it reads this
  // kernel's rows only after its own wait
  pdl_wait();
  pdl_trigger();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int4* col = reinterpret_cast<int4*>(prefix) + blockIdx.x;
  int4 carry = make_int4(0, 0, 0, 0);
  for (int base = 1; base <= n_rows; base += 1024) {
    const int r = base + tid;
    int4 v = (r <= n_rows) ? __ldcg(col + (size_t)r * CG) : make_int4(0, 0, 0, 0);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int x = __shfl_up_sync(kFullMask, v.x, o), y = __shfl_up_sync(kFullMask, v.y, o);
      const int z = __shfl_up_sync(kFullMask, v.z, o), w = __shfl_up_sync(kFullMask, v.w, o);
      if (lane >= o) { v.x += x; v.y += y; v.z += z; v.w += w; }
    }
    if (lane == 31) wsum[warp] = v;
    __syncthreads();
    if (warp == 0) {
      int4 t = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int x = __shfl_up_sync(kFullMask, t.x, o), y = __shfl_up_sync(kFullMask, t.y, o);
        const int z = __shfl_up_sync(kFullMask, t.z, o), w = __shfl_up_sync(kFullMask, t.w, o);
        if (lane >= o) { t.x += x; t.y += y; t.z += z; t.w += w; }
      }
      wsum[lane] = t;
    }
    __syncthreads();
    if (warp > 0) {
      const int4 p = wsum[warp - 1];
      v.x += p.x; v.y += p.y; v.z += p.z; v.w += p.w;
    }
    v.x += carry.x; v.y += carry.y; v.z += carry.z; v.w += carry.w;
    if (r <= n_rows) col[(size_t)r * CG] = v;
    const int4 tot = wsum[31];
    carry.x += tot.x; carry.y += tot.y; carry.z += tot.z; carry.w += tot.w;
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// Token-sharded path: what crosses GPUs is the count matrix
// Lambda[R][E] (lambda_{r,e}: one row per source rank, 4*E_pad bytes each), not the per-chunk rows.
//   shard_rows_kernel    a shard's rows of Lambda = the sums of its source ranks' chunk counts
//                        (launched programmatically dependent on rank_kernel).
// After the exchange nothing runs between it and the planner: plan_kernel adds up the columns of
// Lambda (Alg. 1 line 2), and lookup_kernel (from_lambda) derives the global rank base of its chunk,
// sum_{r' < r} Lambda[r'][e] + the counts of the source rank's earlier chunks, in its prologue.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(UEP_MAX_E)
shard_rows_kernel(int E_pad, int cpg, int rank0, const int32_t* __restrict__ counts, int32_t* __restrict__ lambda) {
  pdl_trigger();                                // the planner behind this kernel may be placed and run its static
                                                // set-up; it lets the lookup start only after its own wait for this grid
  pdl_wait();                                   // shard_hist_kernel complete
  const int r = rank0 + (int)blockIdx.x;
  for (int e = threadIdx.x; e < E_pad; e += blockDim.x) {
    int s = 0;
    for (int q = 0; q < cpg; ++q) s += __ldcg(counts + (size_t)(r * cpg + q) * E_pad + e);
    lambda[(size_t)r * E_pad + e] = s;
  }
}

static void pdl_config(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* attr, dim3 grid, dim3 block, cudaStream_t s, bool pdl) {
  cfg = cudaLaunchConfig_t{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.stream = s;
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
}

int launch_shard_rows(const Ctx* c, void* ws, cudaStream_t s, int rank0, int n_ranks) {
  if (c->S == 0) return UEP_OK;
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(cfg, attr, dim3(n_ranks), dim3(c->E_pad < 32 ? 32 : c->E_pad), s, /*pdl=*/true);
  UEP_CUDA_TRY(cudaLaunchKernelEx(&cfg, shard_rows_kernel, c->E_pad, c->l_cpg, rank0,
                                  (const int32_t*)ws_counts(c, ws), ws_lambda(c, ws)));
  count_launch(c);
  return UEP_OK;
}

// chunk0 / n_launch: the chunk range a token shard owns (uep_shard_count; `ids` is then the
// virtual base of the global [S] array, only the shard's slots are dereferenced); n_launch < 0:
// all chunks.  with_prefix = false leaves the raw per-chunk counts for the exchange step.
// bitmaps = false (uep_balance): the general way.  There the kernel shares its SMs with the planner,
// its end is set by when its second wave of CTAs gets onto the SMs (after the histogram's CTAs
// leave), not by its instruction stream, and the bitmap way's higher issue rate slows the planner's
// probes on the SMs they share (measured, A/B on one box: chain 29.4 -> 29.9 us with it; rank + prefix alone
// 12.3 -> 10.9 us).
int launch_rank(const Ctx* c, const int32_t* ids, void* ws, cudaStream_t s, bool local, int chunk0,
                int n_launch, bool with_prefix, bool bitmaps, bool write_counts) {
  if (c->S == 0) return UEP_OK;
  const int chunks = local ? c->l_chunks : c->r_chunks;
  const int clen = local ? c->l_chunk_len : c->r_chunk_len, k = c->cfg.k;
  const int W = bitmaps ? rank_fast_words(clen, k, c->E_pad) : 0;
  const unsigned k_magic = W > 0 ? 0xffffffffu / (unsigned)k + 1u : 0u;      // ceil(2^32 / k), k >= 2
  const size_t smem = rank_smem_bytes(c->E_pad, W);
  auto kern = W > 0 ? rank_kernel<true> : rank_kernel<false>;
  kern<<<n_launch < 0 ? chunks : n_launch, kRemapThreads, smem, s>>>(
      ids, c->S, c->cfg.E, c->E_pad, clen,
      local ? c->l_cpg : c->r_chunks, local ? c->l_group_len : c->S, ws_packed(c, ws),
      ws_prefix(c, ws), write_counts ? ws_counts(c, ws) : nullptr, chunk0, W, k_magic, write_counts ? 1 : 0);
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  if (with_prefix) return launch_prefix(c, ws, s, local, /*pdl=*/true);
  return UEP_OK;
}

// pdl: launched programmatically dependent on the kernel before it in the stream (rank_kernel):
// the launch latency overlaps that kernel
int launch_prefix(const Ctx* c, void* ws, cudaStream_t s, bool local, bool pdl) {
  if (c->S == 0) return UEP_OK;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(c->E_pad / 4);
  cfg.blockDim = dim3(1024);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  UEP_CUDA_TRY(cudaLaunchKernelEx(&cfg, prefix_kernel, ws_prefix(c, ws),
                                  local ? c->l_chunks : c->r_chunks, c->E_pad / 4));
  count_launch(c);
  return UEP_OK;
}

// ------------------------------------------------------------------------------------------------
// reroute_kernel: SolveReroute, Alg. 1 lines 26-36, one
// WARP per expert.  lambda_{r,e} comes from the prefix table (difference of the rows at the source
// rank's first and last chunk).  Line 29: every host rank first consumes its own quota.  Lines
// 32-34 under reading S18: residual demands (ascending source rank) and residual quotas (instance
// order) are laid on one number line, q[r,e,i] = overlap length (+ the local part): both marginals
// exact, deterministic.  Emits, per source rank r and CSR instance p of the expert,
//   cumq[r][p]   inclusive cumulative of q[r,e,.] in instance order   (the lookup table of §5.2)
//   srcpre[r][p] sum of q[r',e,i] over r' < r                         (receive order: by source rank)
// ------------------------------------------------------------------------------------------------
constexpr int kRrWarps = 4;                        // experts per CTA: one WARP per expert, no block barrier
constexpr int kRrThreads = kRrWarps * 32;
constexpr int kRrMaxInst = UEP_MAX_R + 1;

struct RrWarp {                                    // one warp's tables
  int lamhat[UEP_MAX_R];                           // residual demand of source rank r
  int d0[UEP_MAX_R + 1];                           // its exclusive prefix: the demands' number line
  int host[kRrMaxInst], uhat[kRrMaxInst], loc[kRrMaxInst];
  int u0[kRrMaxInst + 1];                          // exclusive prefix of the residual quotas
  int hidx[UEP_MAX_R];                             // the instance that rank r hosts, -1 = none
};

// exclusive prefix of src[0..n) into dst[0..n], 32 values at a time (dst[n] = total)
__device__ __forceinline__ void rr_warp_excl_scan(const int* src, int* dst, int n, int lane) {
  int carry = 0;
  for (int base = 0; base < n; base += 32) {
    const int v = (base + lane < n) ? src[base + lane] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(kFullMask, inc, o);
      if (lane >= o) inc += y;
    }
    if (base + lane < n) dst[base + lane] = carry + inc - v;
    carry += __shfl_sync(kFullMask, inc, 31);
  }
  if (lane == 0) dst[n] = carry;
}

// (The first version gave an expert a CTA of 256 threads: five block barriers, two block scans and
// running sums over the R source ranks per instance and over the instances per rank — 6.7 us for 0.4 MB.)
__global__ void __launch_bounds__(kRrThreads)
reroute_kernel(int E, int E_pad, int R, int inst_cap, int cpg, const int32_t* __restrict__ prefix,
               const int32_t* __restrict__ inst_off, const int32_t* __restrict__ inst_rank,
               const int32_t* __restrict__ inst_cum, int32_t* __restrict__ cumq,
               int32_t* __restrict__ srcpre, int32_t* __restrict__ n_inflight) {
  __shared__ RrWarp tab[kRrWarps];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = (int)blockIdx.x * kRrWarps + warp;
  pdl_trigger();                 // the lookup's plan-independent prologue may start
  if (e >= E) return;
  RrWarp& w = tab[warp];
  const int lo = inst_off[e], n = inst_off[e + 1] - lo;
  if (e == 0 && n_inflight) for (int r = lane; r < R; r += 32) n_inflight[r] = 0;
  for (int r = lane; r < R; r += 32) {
    w.lamhat[r] = __ldcg(prefix + (size_t)(r + 1) * cpg * E_pad + e) - __ldcg(prefix + (size_t)r * cpg * E_pad + e);
    w.hidx[r] = -1;
  }
  for (int i = lane; i < n; i += 32) {
    w.host[i] = inst_rank[lo + i];
    w.uhat[i] = inst_cum[lo + i] - (i ? inst_cum[lo + i - 1] : 0);
  }
  __syncwarp();
  for (int i = lane; i < n; i += 32) {                       // line 29: consume local quota
    const int h = w.host[i];                                 // (hosts of one expert are distinct ranks)
    const int l = min(w.lamhat[h], w.uhat[i]);
    w.loc[i] = l;
    w.uhat[i] -= l;
    w.lamhat[h] -= l;
    w.hidx[h] = i;
  }
  __syncwarp();
  rr_warp_excl_scan(w.lamhat, w.d0, R, lane);                // number lines (exclusive prefixes)
  rr_warp_excl_scan(w.uhat, w.u0, n, lane);
  __syncwarp();
  // Both tables in closed form, an entry (r, i) per lane and step, no sum left to run: the overlaps
  // of consecutive intervals add up to the overlap with their union,
  //   sum_{i' <= i} q[r,e,i'] = |[d0[r], d0[r+1]) n [0, u0[i+1])|  + the local part if r hosts an instance <= i
  //   sum_{r' <  r} q[r',e,i] = |[0, d0[r])       n [u0[i], u0[i+1])| + the local part if the host of i is below r
  for (int i = 0; i < n; ++i) {
    const int a0 = w.u0[i], a1 = w.u0[i + 1], hi = w.host[i], li = w.loc[i];
    for (int r = lane; r < R; r += 32) {
      const int dr = w.d0[r], dn = w.d0[r + 1], hx = w.hidx[r];
      cumq[(size_t)r * inst_cap + lo + i] = min(max(a1, dr), dn) - dr + ((hx >= 0 && hx <= i) ? w.loc[hx] : 0);
      srcpre[(size_t)r * inst_cap + lo + i] = min(max(dr, a0), a1) - a0 + (hi < r ? li : 0);
    }
  }
}

int launch_reroute(const Ctx* c, const uep_plan_out& plan, int32_t* n_inflight, void* ws, cudaStream_t s) {
  if (c->S == 0) return UEP_OK;
  const int inst_cap = c->cfg.E + c->cfg.R * c->cfg.n_slot;
  int32_t* cumq = ws_reroute(c, ws);
  reroute_kernel<<<(c->cfg.E + kRrWarps - 1) / kRrWarps, kRrThreads, 0, s>>>(c->cfg.E, c->E_pad, c->cfg.R, inst_cap, c->l_cpg, ws_prefix(c, ws),
                                                plan.inst_off, plan.inst_rank, plan.inst_cum, cumq,
                                                cumq + (size_t)c->cfg.R * inst_cap, n_inflight);
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

// ------------------------------------------------------------------------------------------------
// lookup_kernel.  One CTA per chunk, a thread handles kLkPairs PAIRS of consecutive slots (8-byte
// loads and stores).  Everything that does not need the plan runs BEFORE griddepcontrol.wait (under
// programmatic dependent launch it overlaps the planner): the loads of the packed ranks and gates,
// the exclusive prefix el[e] of the chunk's per-expert counts (from rank_kernel's `counts` row),
// and the staging of the gates in (expert, rank) order — a slot's staging position el[e] + rank in
// chunk does not depend on the plan.  After the wait a CTA stages the plan, builds two 8-byte
// records per expert for the instance that holds the chunk's first slot of that expert,
//   rec[e]  = {db, thr << 17 | replica << 8 | rank}   offset = db + jl          while jl < thr
//   grec[e] = {gbx, el[e] + thr}                      out_gate index = gbx + staged position
// and makes two passes: slots in slot order (one random 8-byte record load, three coalesced 8-byte
// stores per pair) and gates in staged order (consecutive positions of an expert go to consecutive
// destinations: coalesced runs).  A slot or gate beyond the first instance's window walks the
// expert's cumulative quotas.  (The first version staged {gate, destination} AFTER the wait with a
// random 8-byte shared store per slot and used 16-byte records: 39 warp instructions per slot,
// 11.5 us between the end of the planner and the last CTA at the DeepSeek-V3 shape.)
// dynamic shared memory layout (ints):
//   rec[E_pad] (int2) | grec[E_pad] (int2) | base0[E_pad] | el[E_pad+4] | s_off[E_pad+4]
//   | rbase[(R+7)&~3] | i_cum | i_base | i_rank (icap each) | wtot[36] | (GATE) stg[kMaxChunk] (int2 {gate bits, e})
// ------------------------------------------------------------------------------------------------
constexpr int kLkPairs = kMaxChunk / 2 / kRemapThreads;       // pairs of slots per thread (8)
constexpr int kLkThrMax = (1 << 14) - 1;                      // thr field of rec: 14 bits, > any rank in a chunk

__host__ __device__ inline size_t lookup_smem_ints(int E_pad, int R, int inst_cap) {
  return 2 * (size_t)E_pad + 2 * (size_t)E_pad + (size_t)E_pad + 2 * (size_t)(E_pad + 4) + ((R + 7) & ~3) +
         3 * (size_t)((inst_cap + 3) & ~3) + 36;           // a multiple of 4: stg is 16-B aligned
}
__host__ __device__ inline size_t lookup_smem_bytes(int E_pad, int R, int inst_cap, bool stage) {
  return sizeof(int) * lookup_smem_ints(E_pad, R, inst_cap) + (stage ? sizeof(int2) * (size_t)kMaxChunk : 0);
}

__device__ __forceinline__ int ld_cg_i32(const int32_t* p) { return __ldcg(p); }

template <typename GateT, bool STAGE, bool LOCAL>
__global__ void __launch_bounds__(kRemapThreads, 2)
lookup_kernel(const int32_t* __restrict__ packed, const GateT* __restrict__ gate, int S, int E,
              int E_pad, int R, int inst_cap, int chunk_len, const int32_t* __restrict__ prefix,
              const int32_t* __restrict__ counts,
              const int32_t* __restrict__ g_inst_off, const int32_t* __restrict__ g_inst_rank,
              const int32_t* __restrict__ g_inst_cum, const int32_t* __restrict__ g_inst_base,
              const int32_t* __restrict__ g_rank_base, int32_t* __restrict__ out_replica,
              int32_t* __restrict__ out_rank, int32_t* __restrict__ out_offset,
              GateT* __restrict__ out_gate, int cpg, int group_len,
              const int32_t* __restrict__ cumq, const int32_t* __restrict__ srcpre,
              int32_t* __restrict__ n_inflight, int32_t* __restrict__ acc_clear, int chunk0,
              const int32_t* __restrict__ lambda) {
  // Token-sharded mode (LOCAL with cumq == nullptr): the grouped chunk geometry and
  // the per-source in-flight count of the source-aware mode, but GLOBAL ranks and the plan's own
  // cumulative quotas, on the chunks [chunk0, chunk0 + gridDim.x) that this GPU owns.
  // Source-aware mode (LOCAL): a group of cpg chunks is one source rank r;
  // ranks are LOCAL to (r, e): base0 = prefix row of the chunk - prefix row of the group's first
  // chunk, the cumulative quotas are row r of cumq (the split q[r,e,.] of SolveReroute) and an
  // instance's base is inst_base + srcpre[r][.] (receive order: by source rank).  Everything else
  // is the same lookup.
  extern __shared__ __align__(16) int smem[];
  int2* rec = reinterpret_cast<int2*>(smem);                 // [E_pad] slot-pass record per expert
  int2* grec = rec + E_pad;                                  // [E_pad] gate-pass record per expert
  int* base0 = reinterpret_cast<int*>(grec + E_pad);         // [E_pad] rank (plan numbering) of the chunk's first slot of e
  int* el = base0 + E_pad;                                   // [E_pad+4] exclusive prefix of the chunk's counts over experts
  int* s_off = el + E_pad + 4;                               // [E_pad+4] CSR of instances
  int* rbase = s_off + E_pad + 4;                            // [(R+7)&~3] rank_base
  const int icap = (inst_cap + 3) & ~3;
  int* i_cum = rbase + ((R + 7) & ~3);           // cumulative quotas (row of the source rank when local)
  int* i_base = i_cum + icap;                    // inst_base (+ srcpre when local)
  int* i_rank = i_base + icap;
  int* wtot = i_rank + icap;                     // [32] warp totals
  int2* stg = reinterpret_cast<int2*>(wtot + 36);     // staged {gate bits, expert}, (expert, rank) order

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c = LOCAL ? (int)blockIdx.x + chunk0 : (int)blockIdx.x;
  const bool local = LOCAL && cumq != nullptr;   // ranks local to (source rank, expert)
  const int grp = LOCAL ? c / cpg : 0, sub = LOCAL ? c % cpg : c;
  const long long cbegin = (long long)grp * group_len + (long long)sub * chunk_len;
  const int clen = LOCAL ? (int)min(min((long long)chunk_len, (long long)group_len - (long long)sub * chunk_len),
                                    (long long)S - cbegin)
                         : (int)min((long long)chunk_len, (long long)S - cbegin);
  const bool has_gate = STAGE && gate != nullptr;
  const bool even = (cbegin & 1) == 0;           // pairs are 8-byte aligned (always, unless a source rank's block is odd)
  packed += cbegin; out_replica += cbegin; out_rank += cbegin; out_offset += cbegin;
  if (has_gate) gate += cbegin;

  // ---- plan-independent prologue ---------------------------------------------------------------
  int2 pv[kLkPairs];
  GateT gv[kLkPairs][2];
#pragma unroll
  for (int it = 0; it < kLkPairs; ++it) {
    const int s0 = 2 * (it * kRemapThreads + tid);
    pv[it] = make_int2(-1, -1);
    if (s0 + 1 < clen && even) {
      pv[it] = __ldcg(reinterpret_cast<const int2*>(packed + s0));
    } else {
      if (s0 < clen) pv[it].x = __ldcg(packed + s0);
      if (s0 + 1 < clen) pv[it].y = __ldcg(packed + s0 + 1);
    }
    if (has_gate) {
      gv[it][0] = s0 < clen ? __ldg(gate + s0) : GateT(0);
      gv[it][1] = s0 + 1 < clen ? __ldg(gate + s0 + 1) : GateT(0);
    }
  }
  // el[e]: exclusive prefix over experts of this chunk's counts (one thread per expert: E <= kRemapThreads)
  {
    const int n_own = (tid < E) ? __ldcg(counts + (size_t)c * E_pad + tid) : 0;
    int inc = n_own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(kFullMask, inc, o);
      if (lane >= o) inc += y;
    }
    if (lane == 31) wtot[warp] = inc;
    __syncthreads();
    int pre = 0;
    for (int w = 0; w < warp; ++w) pre += wtot[w];
    if (tid < E) el[tid] = pre + inc - n_own;
    if (tid == kRemapThreads - 1) el[E] = pre + inc;              // valid slots in this chunk (E < kRemapThreads or == : tid 511 holds the total)
  }
  __syncthreads();
  // token-sharded path: global rank of the chunk's first slot of e = the slots of e on lower source
  // ranks (rows of the gathered Lambda; complete before the planner in front of this kernel started:
  // neither the all-gather nor shard_rows_kernel triggers early) + those in the source rank's earlier
  // chunks (own counts); no prefix kernel.  (Summing the counts of ALL earlier chunks of the shard
  // instead — up to 292 dependent L2 loads per thread on one GPU — took longer than the planner.)
  int p_lam = 0;
  if (LOCAL && lambda != nullptr && tid < E) {
#pragma unroll 8
    for (int r = 0; r < grp; ++r) p_lam += __ldcg(lambda + (size_t)r * E_pad + tid);
    for (int q = 0; q < sub; ++q) p_lam += __ldcg(counts + (size_t)(grp * cpg + q) * E_pad + tid);
  }
  if (has_gate) {                                            // gates into (expert, rank) order
#pragma unroll
    for (int it = 0; it < kLkPairs; ++it) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int pk = u ? pv[it].y : pv[it].x;
        if (pk >= 0) {
          const int e = pk & kEMask;
          stg[el[e] + (pk >> kPackedEBits)] = make_int2((int)gv[it][u], e);
        }
      }
    }
  }

  // ---- everything above is independent of the plan and of prefix_kernel (rank_kernel's outputs were
  // complete before prefix_kernel started); now wait for the planner / prefix_kernel ------------------
  pdl_wait();
  // chunk base ranks: row c of the exclusive prefix over chunks that prefix_kernel left.  Read AFTER
  // the wait, in the same L2 round trip as the plan: under stream capture the lookup's programmatic
  // attribute makes its edge from prefix_kernel programmatic too, and only the wait guarantees that
  // kernel's writes are visible.
  const int p_own = (LOCAL && lambda != nullptr) ? p_lam : (tid < E) ? __ldcg(prefix + (size_t)c * E_pad + tid) : 0;
  const int b0_own = (local && tid < E) ? p_own - __ldcg(prefix + (size_t)grp * cpg * E_pad + tid) : p_own;
  // uep_balance: the planner (now complete) has consumed the histogram's accumulator; clear it for
  // the next call
  if (acc_clear && c == 0) for (int e = tid; e < E; e += kRemapThreads) acc_clear[e] = 0;
  for (int e = tid; e <= E; e += kRemapThreads) s_off[e] = g_inst_off[e];
  for (int r = tid; r <= R; r += kRemapThreads) rbase[r] = g_rank_base[r];
  for (int p = tid; p < inst_cap; p += kRemapThreads) {
    i_cum[p] = local ? __ldcg(cumq + (size_t)grp * inst_cap + p) : g_inst_cum[p];
    i_rank[p] = g_inst_rank[p];
    i_base[p] = g_inst_base[p] + (local ? __ldcg(srcpre + (size_t)grp * inst_cap + p) : 0);
  }
  __syncthreads();
  if (tid < E) {
    const int lo = s_off[tid], last = s_off[tid + 1] - 1, b0 = b0_own;
    int p = lo;
    while (p < last && i_cum[p] <= b0) ++p;
    const int rk = i_rank[p];
    const int d = i_base[p] - (p > lo ? i_cum[p - 1] : 0) + b0;     // offset = d + rank in chunk
    const int thr = min(i_cum[p] - b0, kLkThrMax);                  // ... while rank in chunk < thr
    const int e0 = el[tid];
    base0[tid] = b0;
    rec[tid] = make_int2(d, (int)(((unsigned)thr << 17) | (unsigned)((p - lo) << 8) | (unsigned)rk));
    grec[tid] = make_int2(rbase[rk] + d - e0, e0 + thr);
  }
  __syncthreads();

  // a slot of expert e with rank jl in the chunk that lies beyond the first instance's window
  auto walk = [&](int e, int jl, int rep0, int& rep, int& rk, int& db) {
    const int b0 = base0[e], j = jl + b0;
    int p = s_off[e] + rep0 + 1;
    const int last = s_off[e + 1] - 1;             // cum[last] = lambda_e > j when ws matches plan
    while (p < last && i_cum[p] <= j) ++p;
    rk = i_rank[p];
    db = i_base[p] - i_cum[p - 1] + b0;            // p > s_off[e]: cum_prev is the entry before
    rep = p - s_off[e];
  };

  // ---- slot pass ----------------------------------------------------------------------------------
  int n_fly = 0;
#pragma unroll
  for (int it = 0; it < kLkPairs; ++it) {
    const int s0 = 2 * (it * kRemapThreads + tid);
    if (s0 < clen) {
      int rep[2], rk[2], of[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int pk = u ? pv[it].y : pv[it].x;
        rep[u] = -1; rk[u] = -1; of[u] = -1;
        if (pk >= 0) {
          const int e = pk & kEMask, jl = pk >> kPackedEBits;
          const int2 rc = rec[e];
          const unsigned w = (unsigned)rc.y;
          int db = rc.x;
          rep[u] = (int)((w >> 8) & 0x1ffu);
          rk[u] = (int)(w & 0xffu);
          if (jl >= (int)(w >> 17)) walk(e, jl, rep[u], rep[u], rk[u], db);
          of[u] = db + jl;
          if (LOCAL) n_fly += (rk[u] != grp) ? 1 : 0;
        }
      }
      if (s0 + 1 < clen && even) {
        *reinterpret_cast<int2*>(out_replica + s0) = make_int2(rep[0], rep[1]);
        *reinterpret_cast<int2*>(out_rank + s0) = make_int2(rk[0], rk[1]);
        *reinterpret_cast<int2*>(out_offset + s0) = make_int2(of[0], of[1]);
      } else {
        out_replica[s0] = rep[0]; out_rank[s0] = rk[0]; out_offset[s0] = of[0];
        if (s0 + 1 < clen) { out_replica[s0 + 1] = rep[1]; out_rank[s0 + 1] = rk[1]; out_offset[s0 + 1] = of[1]; }
      }
    }
  }
  if (LOCAL && n_inflight) {                             // tokens of source rank grp that leave it
    n_fly = __reduce_add_sync(kFullMask, n_fly);
    if (lane == 0 && n_fly) atomicAdd(n_inflight + grp, n_fly);
  }

  // ---- gate pass: staged order, consecutive positions of an expert go to consecutive destinations ---
  if (has_gate) {
    const int n_valid = el[E];
#pragma unroll 4
    for (int ps = tid; ps < n_valid; ps += kRemapThreads) {
      const int2 v = stg[ps];
      const int2 g = grec[v.y];
      int dst = g.x + ps;
      if (ps >= g.y) {                                   // beyond the first instance's window
        const int e = v.y, jl = ps - el[e];
        int rep, rk, db;
        walk(e, jl, (int)(((unsigned)rec[e].y >> 8) & 0x1ffu), rep, rk, db);
        dst = rbase[rk] + db + jl;
      }
      out_gate[dst] = (GateT)v.x;
    }
  }
}

template <typename GateT>
static int launch_lookup_t(const Ctx* c, const GateT* gate, const uep_plan_out& p,
                           int32_t* out_replica, int32_t* out_rank, int32_t* out_offset,
                           GateT* out_gate, void* ws, cudaStream_t s, bool pdl, bool local,
                           int32_t* n_inflight, int32_t* acc_clear, int chunk0, int n_launch,
                           bool src_aware, bool from_lambda) {
  const uep_config& g = c->cfg;
  const int inst_cap = g.E + g.R * g.n_slot;
  const bool stage = gate != nullptr;
  const size_t smem = lookup_smem_bytes(c->E_pad, g.R, inst_cap, stage);
  auto k = local ? (stage ? lookup_kernel<GateT, true, true> : lookup_kernel<GateT, false, true>)
                 : (stage ? lookup_kernel<GateT, true, false> : lookup_kernel<GateT, false, false>);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(n_launch >= 0 ? n_launch : (local ? c->l_chunks : c->r_chunks));
  cfg.blockDim = dim3(kRemapThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  const int32_t* cumq = (local && src_aware) ? ws_reroute(c, ws) : nullptr;
  const int32_t* srcpre = cumq ? cumq + (size_t)g.R * inst_cap : nullptr;
  UEP_CUDA_TRY(cudaLaunchKernelEx(&cfg, k, (const int32_t*)ws_packed(c, ws), gate, c->S, g.E, c->E_pad,
                                  g.R, inst_cap, local ? c->l_chunk_len : c->r_chunk_len,
                                  (const int32_t*)ws_prefix(c, ws), (const int32_t*)ws_counts(c, ws),
                                  (const int32_t*)p.inst_off, (const int32_t*)p.inst_rank,
                                  (const int32_t*)p.inst_cum, (const int32_t*)p.inst_base,
                                  (const int32_t*)p.rank_base, out_replica, out_rank, out_offset,
                                  out_gate, local ? c->l_cpg : c->r_chunks, local ? c->l_group_len : c->S,
                                  cumq, srcpre, n_inflight, acc_clear, chunk0,
                                  from_lambda ? (const int32_t*)ws_lambda(c, ws) : (const int32_t*)nullptr));
  count_launch(c);
  return UEP_OK;
}

int init_remap_kernels() {
  int rc = prefer_max_smem(rank_kernel<false>);
  if (rc == UEP_OK) rc = prefer_max_smem(rank_kernel<true>);
  if (rc == UEP_OK) rc = prefer_max_smem(prefix_kernel);
  if (rc == UEP_OK) rc = prefer_max_smem(reroute_kernel);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint32_t, true, false>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint32_t, true, true>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint32_t, false, false>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint32_t, false, true>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint16_t, true, false>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint16_t, true, true>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint16_t, false, false>);
  if (rc == UEP_OK) rc = prefer_max_smem(lookup_kernel<uint16_t, false, true>);
  if (rc != UEP_OK) return rc;
  const int rank_bytes = (int)std::max(sizeof(int2) * (size_t)kRemapWarps * UEP_MAX_E, kRankFastSmem + 16);
  const int bytes = (int)lookup_smem_bytes(UEP_MAX_E, UEP_MAX_R, UEP_MAX_E + UEP_MAX_R * UEP_MAX_NSLOT, true);
  UEP_CUDA_TRY(cudaFuncSetAttribute(rank_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, rank_bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(rank_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, rank_bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint32_t, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint32_t, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint32_t, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint32_t, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint16_t, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint16_t, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint16_t, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  UEP_CUDA_TRY(cudaFuncSetAttribute(lookup_kernel<uint16_t, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  return UEP_OK;
}

int launch_lookup(const Ctx* c, const void* gate, const uep_plan_out& p, int32_t* out_replica,
                  int32_t* out_rank, int32_t* out_offset, void* out_gate, void* ws, cudaStream_t s,
                  bool pdl, bool local, int32_t* n_inflight, int32_t* acc_clear, int chunk0,
                  int n_launch, bool src_aware, bool from_lambda) {
  if (c->S == 0) return UEP_OK;
  if (c->cfg.gate_dtype == UEP_GATE_BF16 && gate)
    return launch_lookup_t<uint16_t>(c, static_cast<const uint16_t*>(gate), p, out_replica, out_rank,
                                     out_offset, static_cast<uint16_t*>(out_gate), ws, s, pdl, local, n_inflight, acc_clear,
                                     chunk0, n_launch, src_aware, from_lambda);
  return launch_lookup_t<uint32_t>(c, static_cast<const uint32_t*>(gate), p, out_replica, out_rank,
                                   out_offset, static_cast<uint32_t*>(out_gate), ws, s, pdl, local, n_inflight, acc_clear,
                                   chunk0, n_launch, src_aware, from_lambda);
}

int launch_remap(const Ctx* c, const int32_t* ids, const void* gate, const uep_plan_out& p,
                 int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                 void* ws, cudaStream_t s) {
  int rc = launch_rank(c, ids, ws, s);
  if (rc != UEP_OK) return rc;
  // programmatically dependent on prefix_kernel: launch and the loads of packed ranks and gates
  // overlap it, the prefix rows are read after the wait
  return launch_lookup(c, gate, p, out_replica, out_rank, out_offset, out_gate, ws, s, /*pdl=*/true);
}

}  // namespace uep
