// hist.cu — uep_histogram: lambda_e = #{s : topk_ids[s] == e}  (Alg. 1 line 2).
//
// HBM-bound: 4 B/slot read once.  One CTA per chunk (one chunk per SM).  Every thread issues
// all of its int4 loads of a round before it touches shared memory (kHistVecs x 16 B in flight
// per thread, 64 KB per SM), then counts into a WARP-PRIVATE shared-memory row (pitch E_pad+1
// so the same expert in different rows falls into different banks): no contention between
// warps on a hot expert, only the intra-warp multiplicity.  The CTA's row of the chunk table
// (raw counts, used only by this kernel's own reduction) is written once.  The last
// CTA to finish (ticket) sums the table's columns with one round of independent int4 L2 loads
// and emits expert_count.  Integer adds only: bit-identical run to run.
#include "uep_internal.cuh"

namespace uep {

constexpr int kHistWarps = kHistThreads / 32;
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

// dynamic shared memory (ints): priv[kHistWarps][E_pad+1] | part[kColPartInts] | tot[E_pad]
__host__ __device__ inline size_t hist_smem_ints(int E_pad) {
  return (size_t)kHistWarps * (E_pad + 1) + kColPartInts + E_pad;
}

// RED = false: the CTA's row goes to the chunk table, the last CTA (ticket) sums the columns into
// expert_count.  RED = true (uep_balance): the ticket, the fence and the last CTA's serial pass cost
// 4.8 of the kernel's 9.4 us at the DeepSeek-V3 shape, so every CTA instead adds its counts to an
// accumulator in the workspace with fire-and-forget reductions (integer adds: order-free) and
// exits; the planner reads the accumulator, publishes expert_count and clears it.
template <bool RED>
__global__ void __launch_bounds__(kHistThreads, 1)
hist_kernel(const int32_t* __restrict__ ids, int S, int E, int E_pad, int chunk_len,
            int n_chunks, int32_t* __restrict__ table, unsigned* __restrict__ ticket,
            int32_t* __restrict__ expert_count) {
  extern __shared__ __align__(16) int hsm[];
  const int pitch = E_pad + 1;
  int* priv = hsm;
  int* part = hsm + ((kHistWarps * pitch + 3) & ~3);
  int* tot = part + kColPartInts;
  __shared__ unsigned s_last;
  const int tid = threadIdx.x, warp = tid >> 5;
  const int c = blockIdx.x;
  pdl_trigger();     // uep_balance launches the planner behind this kernel with its prologue overlapped

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
  for (int i = tid; i < kHistWarps * pitch; i += kHistThreads) priv[i] = 0;
  __syncthreads();

  int* row = priv + warp * pitch;
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

  int32_t* grow = table + (size_t)c * E_pad;
  for (int e = tid; e < E_pad; e += kHistThreads) {
    int s = 0;
#pragma unroll 8
    for (int w = 0; w < kHistWarps; ++w) s += priv[w * pitch + e];
    if (RED) { if (s != 0 && e < E) atomicAdd(expert_count + e, s); }   // expert_count = the accumulator
    else grow[e] = s;
  }
  if (RED) return;
  __syncthreads();                   // the CTA's row is written (barrier orders it before thread 0's fence)
  if (tid == 0) {
    __threadfence();                 // cumulative: makes the whole row visible before the ticket
    s_last = (atomicAdd(ticket, 1u) == (unsigned)(n_chunks - 1));
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();

  // Last CTA: column totals -> expert_count.
  column_sums(table, n_chunks, E_pad, part, tot);
  for (int e = tid; e < E; e += kHistThreads) expert_count[e] = tot[e];
  if (tid == 0) *ticket = 0u;        // self-reset: the next launch (graph replay) starts clean
}

// S == 0: nothing to read; zero the counts and the single table row.
__global__ void hist_empty_kernel(int E, int E_pad, int32_t* table, int32_t* expert_count) {
  for (int e = threadIdx.x; e < E_pad; e += blockDim.x) {
    table[e] = 0;
    if (e < E) expert_count[e] = 0;
  }
}

int init_hist_kernels() {
  UEP_CUDA_TRY(cudaFuncSetAttribute(hist_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(int) * (hist_smem_ints(UEP_MAX_E) + 4))));
  UEP_CUDA_TRY(cudaFuncSetAttribute(hist_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(int) * (hist_smem_ints(UEP_MAX_E) + 4))));
  return UEP_OK;
}

int launch_histogram(const Ctx* c, const int32_t* ids, int32_t* count, void* ws, cudaStream_t s,
                     bool red) {
  if (c->S == 0) {
    if (!red) hist_empty_kernel<<<1, 256, 0, s>>>(c->cfg.E, c->E_pad, ws_table(ws), count);
  } else {
    const size_t smem = sizeof(int) * (hist_smem_ints(c->E_pad) + 4);
    if (red)
      hist_kernel<true><<<c->n_chunks, kHistThreads, smem, s>>>(ids, c->S, c->cfg.E, c->E_pad,
                                                                c->chunk_len, c->n_chunks, ws_table(ws),
                                                                ws_ticket(ws), ws_acc(ws));
    else
      hist_kernel<false><<<c->n_chunks, kHistThreads, smem, s>>>(ids, c->S, c->cfg.E, c->E_pad,
                                                                 c->chunk_len, c->n_chunks, ws_table(ws),
                                                                 ws_ticket(ws), count);
  }
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

}  // namespace uep
