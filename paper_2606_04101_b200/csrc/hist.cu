// hist.cu — uep_histogram: lambda_e = #{s : topk_ids[s] == e}  (Alg. 1 line 2).
//
// HBM-bound: 4 B/slot read once.  One CTA per chunk (one chunk per SM), int4-vectorised
// coalesced loads issued up front, a per-CTA shared-memory histogram (E <= 512), one row of
// the chunk table written per CTA.  The last CTA to finish (ticket) turns the table into its
// exclusive prefix over chunks — what uep_remap needs for global stable ranks — and emits the
// column totals as expert_count.  No float, no order-dependent atomics: results are
// bit-identical run to run.
#include "uep_internal.cuh"

namespace uep {

__device__ __forceinline__ int4 ld_stream_v4(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

__device__ __forceinline__ void count_one(int* hist, int e, int E) {
  if ((unsigned)e < (unsigned)E) atomicAdd(&hist[e], 1);
}

constexpr int kHistUnroll = 4;

__global__ void __launch_bounds__(kHistThreads, 1)
hist_kernel(const int32_t* __restrict__ ids, int S, int E, int E_pad, int chunk_len,
            int n_chunks, int32_t* __restrict__ table, unsigned* __restrict__ ticket,
            int32_t* __restrict__ expert_count) {
  __shared__ int hist[UEP_MAX_E];
  __shared__ int part[kHistThreads];
  __shared__ unsigned s_last;
  const int tid = threadIdx.x;
  const int c = blockIdx.x;
  for (int e = tid; e < E_pad; e += kHistThreads) hist[e] = 0;
  __syncthreads();

  const long long begin = (long long)c * chunk_len;
  const int len = (int)min((long long)chunk_len, (long long)S - begin);   // > 0 by construction
  const int n_vec = len >> 2;
  const int4* v = reinterpret_cast<const int4*>(ids + begin);             // chunk_len % 128 == 0
  int i = tid;
  for (; i + (kHistUnroll - 1) * kHistThreads < n_vec; i += kHistUnroll * kHistThreads) {
    int4 x[kHistUnroll];
#pragma unroll
    for (int u = 0; u < kHistUnroll; ++u) x[u] = ld_stream_v4(v + i + u * kHistThreads);
#pragma unroll
    for (int u = 0; u < kHistUnroll; ++u) {
      count_one(hist, x[u].x, E); count_one(hist, x[u].y, E);
      count_one(hist, x[u].z, E); count_one(hist, x[u].w, E);
    }
  }
  for (; i < n_vec; i += kHistThreads) {
    int4 x = ld_stream_v4(v + i);
    count_one(hist, x.x, E); count_one(hist, x.y, E);
    count_one(hist, x.z, E); count_one(hist, x.w, E);
  }
  if (tid < (len & 3)) count_one(hist, ids[begin + (n_vec << 2) + tid], E);   // ragged tail
  __syncthreads();

  int32_t* row = table + (size_t)c * E_pad;
  for (int e = tid; e < E_pad; e += kHistThreads) row[e] = hist[e];
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(ticket, 1u) == (unsigned)(n_chunks - 1));
  __syncthreads();
  if (!s_last) return;
  __threadfence();

  // Last CTA: exclusive prefix over chunks, per expert column; totals -> expert_count.
  // G thread groups split the rows; each (column, group) thread walks its row segment.
  const int G = max(1, min(kHistThreads / E_pad, n_chunks));
  const int seg = (n_chunks + G - 1) / G;
  const int col = tid % E_pad, g = tid / E_pad;
  const bool act = (tid < E_pad * G);
  const int r0 = g * seg, r1 = min(n_chunks, r0 + seg);
  int sum = 0;
  if (act) {
#pragma unroll 8
    for (int r = r0; r < r1; ++r) sum += __ldcg(table + (size_t)r * E_pad + col);
    part[tid] = sum;
  }
  __syncthreads();
  if (act) {
    int run = 0;
    for (int gg = 0; gg < g; ++gg) run += part[gg * E_pad + col];
#pragma unroll 8
    for (int r = r0; r < r1; ++r) {
      int32_t* p = table + (size_t)r * E_pad + col;
      const int x = __ldcg(p);
      *p = run;
      run += x;
    }
    if (g == G - 1 && col < E) expert_count[col] = run;
  }
  if (tid == 0) *ticket = 0u;        // self-reset: the next launch (graph replay) starts clean
}

// S == 0: nothing to read; zero the counts and the single table row.
__global__ void hist_empty_kernel(int E, int E_pad, int32_t* table, int32_t* expert_count) {
  for (int e = threadIdx.x; e < E_pad; e += blockDim.x) {
    table[e] = 0;
    if (e < E) expert_count[e] = 0;
  }
}

int launch_histogram(const Ctx* c, const int32_t* ids, int32_t* count, void* ws, cudaStream_t s) {
  if (c->S == 0) {
    hist_empty_kernel<<<1, 256, 0, s>>>(c->cfg.E, c->E_pad, ws_table(ws), count);
  } else {
    hist_kernel<<<c->n_chunks, kHistThreads, 0, s>>>(ids, c->S, c->cfg.E, c->E_pad, c->chunk_len,
                                                     c->n_chunks, ws_table(ws), ws_ticket(ws), count);
  }
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

}  // namespace uep
