// hist.cu — uep_histogram: lambda_e = #{s : topk_ids[s] == e}  (Alg. 1 line 2).
//
// HBM-bound: 4 B/slot read once.  One CTA per chunk (one chunk per SM).  Every thread issues
// all of its int4 loads of a round before it touches shared memory (kHistVecs x 16 B in flight
// per thread, 64 KB per SM), then counts into a shared-memory row that four warps share (8 rows,
// pitch E_pad+1 so the same expert in different rows falls into different banks; shared atomics
// cost ~1.2 cycles per warp instruction and SM on this part, so a row per warp — 32 rows to zero
// and to add up — bought nothing: 5.42 -> 5.31 us with 8).  Every CTA adds its column sums to an
// accumulator in the workspace (zero between calls) with fire-and-forget reductions — integer
// adds, order-free, bit-identical run to run — and exits.  The accumulator is consumed by the
// kernel behind it in the stream, launched programmatically dependent: the planner inside
// uep_balance (it publishes expert_count), publish_kernel in the standalone uep_histogram (one
// CTA: accumulator -> expert_count, accumulator cleared).  An earlier design elected the last CTA
// by a ticket and summed a table of per-CTA rows there: fence + ticket + that CTA's serial pass
// cost 4.8 of the kernel's 9.4 us at the DeepSeek-V3 shape.
#include "uep_internal.cuh"

namespace uep {

constexpr int kHistWarps = kHistThreads / 32;
constexpr int kHistShare = 2;                                 // log2 of the warps sharing a row of counters
constexpr int kHistRows = kHistWarps >> kHistShare;
constexpr int kHistVecs = 4;                                  // int4 loads per thread per round

__device__ __forceinline__ int4 ld_stream_v4(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

__device__ __forceinline__ void count_one(int* row, int e, int E) {
  if ((unsigned)e < (unsigned)E) atomicAdd(&row[e], 1);
}

// dynamic shared memory (ints): priv[kHistRows][E_pad+1]
__host__ __device__ inline size_t hist_smem_ints(int E_pad) {
  return (size_t)kHistRows * (E_pad + 1);
}

// TABLE: also leave the CTA's raw counts in row c of the chunk table (uep_histogram's by-product,
// SURVEY 8(a1); uep_balance does not need it)
template <bool TABLE>
__global__ void __launch_bounds__(kHistThreads, 1)
hist_kernel(const int32_t* __restrict__ ids, int S, int E, int E_pad, int chunk_len,
            int32_t* __restrict__ table, int32_t* __restrict__ acc) {
  extern __shared__ __align__(16) int hsm[];
  const int pitch = E_pad + 1;
  int* priv = hsm;
  const int tid = threadIdx.x, warp = tid >> 5;
  const int c = blockIdx.x;
  pdl_trigger();     // the kernel behind this one (planner / publish_kernel) may start its prologue

  const long long begin = (long long)c * chunk_len;
  const int len = (int)min((long long)chunk_len, (long long)S - begin);   // > 0 by construction
  const int n_vec = len >> 2;
  const int4* v = reinterpret_cast<const int4*>(ids + begin);             // chunk_len % 128 == 0

  // first round's loads go out before the shared-memory rows are zeroed
  int4 x[kHistVecs];
#pragma unroll
  for (int u = 0; u < kHistVecs; ++u) {
    const int i = u * kHistThreads + tid;
    x[u] = (i < n_vec) ? ld_stream_v4(v + i) : make_int4(-1, -1, -1, -1);
  }
  for (int i = tid; i < kHistRows * pitch; i += kHistThreads) priv[i] = 0;
  __syncthreads();

  int* row = priv + (warp >> kHistShare) * pitch;
  for (int vbase = 0; vbase < n_vec; vbase += kHistThreads * kHistVecs) {
#pragma unroll
    for (int u = 0; u < kHistVecs; ++u) {
      count_one(row, x[u].x, E); count_one(row, x[u].y, E);
      count_one(row, x[u].z, E); count_one(row, x[u].w, E);
    }
    const int nb = vbase + kHistThreads * kHistVecs;
    if (nb < n_vec) {
#pragma unroll
      for (int u = 0; u < kHistVecs; ++u) {
        const int i = nb + u * kHistThreads + tid;
        x[u] = (i < n_vec) ? ld_stream_v4(v + i) : make_int4(-1, -1, -1, -1);
      }
    }
  }
  if (tid < (len & 3)) count_one(row, ids[begin + (n_vec << 2) + tid], E);   // ragged tail
  __syncthreads();

  for (int e = tid; e < E_pad; e += kHistThreads) {
    int s = 0;
#pragma unroll 8
    for (int w = 0; w < kHistRows; ++w) s += priv[w * pitch + e];
    if (s != 0 && e < E) atomicAdd(acc + e, s);          // result unused: a fire-and-forget RED
    if (TABLE) table[(size_t)c * E_pad + e] = s;
  }
}

// uep_histogram's second kernel, one CTA, launched programmatically dependent on hist_kernel (its
// launch overlaps it): accumulator -> expert_count, accumulator cleared for the next call.
__global__ void __launch_bounds__(UEP_MAX_E)
publish_kernel(int E, int32_t* __restrict__ acc, int32_t* __restrict__ expert_count) {
  pdl_wait();                        // hist_kernel complete, its reductions performed
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    expert_count[e] = __ldcg(acc + e);
    acc[e] = 0;
  }
}

// Token-sharded path: the count rows of the GROUPED chunks (chunk cb = sub-chunk cb % cpg
// of source rank cb / cpg, never across two source ranks' blocks) without the ranks — the quick half
// of uep_shard_count, so that the rows for the exchange are ready after one pass over the ids while
// rank_kernel works beside it.  Same counting scheme as hist_kernel; a chunk may start anywhere, so the
// 16-byte loads begin at the first aligned slot.  Row cb of `counts` gets the chunk's counts.
constexpr int kShThreads = 512;                               // two CTAs per SM: the 256 chunks of the DeepSeek-V3 shape in one wave
constexpr int kShRows = (kShThreads / 32) >> kHistShare;
__global__ void __launch_bounds__(kShThreads, 2)
shard_hist_kernel(const int32_t* __restrict__ ids, int S, int E, int E_pad, int chunk_len, int cpg,
                  int group_len, int32_t* __restrict__ counts, int chunk0) {
  extern __shared__ __align__(16) int hsm[];
  const int pitch = E_pad + 1;
  int* priv = hsm;
  const int tid = threadIdx.x, warp = tid >> 5;
  const int cb = (int)blockIdx.x + chunk0;
  pdl_trigger();
  const int grp = cb / cpg, sub = cb - grp * cpg;
  const long long cbegin = (long long)grp * group_len + (long long)sub * chunk_len;
  const int clen = (int)min(min((long long)chunk_len, (long long)group_len - (long long)sub * chunk_len),
                            (long long)S - cbegin);
  for (int i = tid; i < kShRows * pitch; i += kShThreads) priv[i] = 0;
  __syncthreads();
  int* row = priv + (warp >> kHistShare) * pitch;
  const int32_t* p = ids + cbegin;
  const int lead = min(clen, (int)(((16u - (unsigned)(reinterpret_cast<uintptr_t>(p) & 15u)) & 15u) >> 2));
  if (tid < lead) count_one(row, p[tid], E);
  const int4* v = reinterpret_cast<const int4*>(p + lead);
  const int n_vec = (clen - lead) >> 2;
  for (int vbase = 0; vbase < n_vec; vbase += kShThreads * kHistVecs) {     // all loads of a round in flight first
    int4 x[kHistVecs];
#pragma unroll
    for (int u = 0; u < kHistVecs; ++u) {
      const int i = vbase + u * kShThreads + tid;
      x[u] = (i < n_vec) ? ld_stream_v4(v + i) : make_int4(-1, -1, -1, -1);
    }
#pragma unroll
    for (int u = 0; u < kHistVecs; ++u) {
      count_one(row, x[u].x, E); count_one(row, x[u].y, E);
      count_one(row, x[u].z, E); count_one(row, x[u].w, E);
    }
  }
  const int t0 = lead + (n_vec << 2);
  if (tid < clen - t0) count_one(row, p[t0 + tid], E);
  __syncthreads();
  for (int e = tid; e < E_pad; e += kShThreads) {
    int s = 0;
#pragma unroll 8
    for (int w = 0; w < kShRows; ++w) s += priv[w * pitch + e];
    counts[(size_t)cb * E_pad + e] = s;
  }
}

// S == 0: nothing to read; zero the counts and the single table row.
__global__ void hist_empty_kernel(int E, int E_pad, int32_t* table, int32_t* expert_count) {
  for (int e = threadIdx.x; e < E_pad; e += blockDim.x) {
    table[e] = 0;
    if (e < E) expert_count[e] = 0;
  }
}

int init_hist_kernels() {
  int rc = prefer_max_smem(hist_kernel<false>);
  if (rc == UEP_OK) rc = prefer_max_smem(hist_kernel<true>);
  if (rc == UEP_OK) rc = prefer_max_smem(publish_kernel);
  if (rc == UEP_OK) rc = prefer_max_smem(shard_hist_kernel);
  if (rc != UEP_OK) return rc;
  UEP_CUDA_TRY(cudaFuncSetAttribute(shard_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(int) * (hist_smem_ints(UEP_MAX_E) + 4))));
  UEP_CUDA_TRY(cudaFuncSetAttribute(hist_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(int) * (hist_smem_ints(UEP_MAX_E) + 4))));
  UEP_CUDA_TRY(cudaFuncSetAttribute(hist_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(int) * (hist_smem_ints(UEP_MAX_E) + 4))));
  return UEP_OK;
}

int launch_shard_hist(const Ctx* c, const int32_t* ids, void* ws, cudaStream_t s, int chunk0, int n_launch) {
  if (c->S == 0 || n_launch <= 0) return UEP_OK;
  const size_t smem = sizeof(int) * (hist_smem_ints(c->E_pad) + 4);
  shard_hist_kernel<<<n_launch, kShThreads, smem, s>>>(ids, c->S, c->cfg.E, c->E_pad, c->l_chunk_len, c->l_cpg,
                                                        c->l_group_len, ws_counts(c, ws), chunk0);
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

// red = true (uep_balance): only the accumulator is left, for the planner.
int launch_histogram(const Ctx* c, const int32_t* ids, int32_t* count, void* ws, cudaStream_t s,
                     bool red) {
  if (c->S == 0) {
    if (!red) hist_empty_kernel<<<1, 256, 0, s>>>(c->cfg.E, c->E_pad, ws_table(ws), count);
    UEP_CUDA_TRY(cudaGetLastError());
    if (!red) count_launch(c);
    return UEP_OK;
  }
  const size_t smem = sizeof(int) * (hist_smem_ints(c->E_pad) + 4);
  if (red) {
    // (launching this kernel programmatically dependent on its predecessor, with a wait at its
    // top, was measured: the 1.5-1.9 us between the end of one call's lookup and the start of the
    // next call's histogram are completion-to-release latency, not launch latency, and stayed)
    hist_kernel<false><<<c->n_chunks, kHistThreads, smem, s>>>(ids, c->S, c->cfg.E, c->E_pad,
                                                               c->chunk_len, ws_table(ws), ws_acc(ws));
    UEP_CUDA_TRY(cudaGetLastError());
    count_launch(c);
    return UEP_OK;
  }
  hist_kernel<true><<<c->n_chunks, kHistThreads, smem, s>>>(ids, c->S, c->cfg.E, c->E_pad,
                                                            c->chunk_len, ws_table(ws), ws_acc(ws));
  UEP_CUDA_TRY(cudaGetLastError());
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1);
  cfg.blockDim = dim3(c->E_pad < 32 ? 32 : c->E_pad);
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  UEP_CUDA_TRY(cudaLaunchKernelEx(&cfg, publish_kernel, c->cfg.E, ws_acc(ws), count));
  count_launch(c, 2);
  return UEP_OK;
}

}  // namespace uep
