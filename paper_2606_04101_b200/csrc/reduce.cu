// reduce.cu — the backward half on one GPU:
//
//   uep_grad_reduce    "every main expert aggregates the gradients contributed by all of its
//                      remote replicas into the main gradient buffer" (§4.2);
//                      "gradient tiles from remote replicas are loaded and accumulated into the
//                      local gradient buffer of main experts, and then cleared in place for reuse
//                      in later layers" (§6.1).  fp32.
//   uep_remap_inverse  the reverse reroute, "a scatter-to-gather inversion of the forward
//                      assignment": src[rank_base[rank]+offset] = slot.
//
// grad_reduce_kernel is HBM-bound: per replicated expert with f replicas it reads (1+f) B and
// writes (1+f) B (the sum, and zeros).  Kept from the paper: fixed tiles, a persistent static grid
// (capturable although the work list is data-dependent), every tile of the main buffer touched
// once.  Each thread owns float4 elements of the tile; the addends are added in instance order
// (main, then replicas in acceptance order), so the fp32 result is bit-identical run to run and
// equal to a sequential fp32 sum in that order.
#include "uep_internal.cuh"

namespace uep {

constexpr int kRedThreads = 512;
constexpr int kRedVec = 4;                                   // float4 per thread per tile
constexpr int kRedTileBytes = kRedThreads * kRedVec * 16;    // 32 KB of fp32 per tile
constexpr int kRedMaxFan = UEP_MAX_R;                        // replicas of one expert

struct RedArgs {
  float* main_grad[UEP_MAX_TENSORS];
  float* slot_grad[UEP_MAX_TENSORS];
  unsigned long long bytes[UEP_MAX_TENSORS];
  int n_tensors;
};

__global__ void __launch_bounds__(kRedThreads, 2)
grad_reduce_kernel(RedArgs a, int E, int n_slot, int M, const int32_t* __restrict__ inst_off,
                   const int32_t* __restrict__ inst_rank, const int32_t* __restrict__ inst_phys) {
  __shared__ int s_slot[kRedMaxFan];
  const int tid = threadIdx.x, G = gridDim.x, c = blockIdx.x;
  unsigned rot = 0;                               // rotation so that tile remainders spread over CTAs
  for (int e = 0; e < E; ++e) {
    const int lo = inst_off[e], f = inst_off[e + 1] - lo - 1;      // f replicas (entry lo = main)
    if (f <= 0) continue;
    __syncthreads();                              // previous expert done with s_slot
    for (int p = tid; p < f; p += kRedThreads)
      s_slot[p] = inst_rank[lo + 1 + p] * n_slot + (inst_phys[lo + 1 + p] - M);
    __syncthreads();
    for (int j = 0; j < a.n_tensors; ++j) {
      const unsigned long long B = a.bytes[j];
      const long long tiles = (long long)((B + kRedTileBytes - 1) / kRedTileBytes);
      float4* mainp = reinterpret_cast<float4*>(reinterpret_cast<unsigned char*>(a.main_grad[j]) +
                                                (unsigned long long)e * B);
      unsigned char* slots = reinterpret_cast<unsigned char*>(a.slot_grad[j]);
      const long long n4 = (long long)(B >> 4);
      for (long long tile = (c + G - (int)rot) % G; tile < tiles; tile += G) {
        const long long base = tile * (kRedTileBytes >> 4);
        float4 acc[kRedVec];
#pragma unroll
        for (int v = 0; v < kRedVec; ++v) {
          const long long i = base + v * kRedThreads + tid;
          acc[v] = (i < n4) ? __ldcs(mainp + i) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        for (int p = 0; p < f; ++p) {             // instance order: main, replica 1, replica 2, ...
          float4* sp = reinterpret_cast<float4*>(slots + (unsigned long long)s_slot[p] * B);
          float4 x[kRedVec];
#pragma unroll
          for (int v = 0; v < kRedVec; ++v) {
            const long long i = base + v * kRedThreads + tid;
            x[v] = (i < n4) ? __ldcs(sp + i) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
#pragma unroll
          for (int v = 0; v < kRedVec; ++v) {
            const long long i = base + v * kRedThreads + tid;
            acc[v].x += x[v].x; acc[v].y += x[v].y; acc[v].z += x[v].z; acc[v].w += x[v].w;
            if (i < n4) __stcs(sp + i, make_float4(0.f, 0.f, 0.f, 0.f));   // cleared in place
          }
        }
#pragma unroll
        for (int v = 0; v < kRedVec; ++v) {
          const long long i = base + v * kRedThreads + tid;
          if (i < n4) __stcs(mainp + i, acc[v]);
        }
      }
      rot = (unsigned)((rot + tiles) % (unsigned)G);
    }
  }
}

__global__ void __launch_bounds__(256)
inverse_kernel(const int32_t* __restrict__ out_rank, const int32_t* __restrict__ out_offset,
               const int32_t* __restrict__ rank_base, int S, int R, int32_t* __restrict__ out_src) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= S) return;
  const int n_valid = __ldg(rank_base + R);
  const int r = __ldg(out_rank + s);
  if (r >= 0) out_src[__ldg(rank_base + r) + __ldg(out_offset + s)] = s;
  if (s >= n_valid) out_src[s] = -1;       // positions past the valid slots (destinations are < n_valid)
}

int launch_grad_reduce(const Ctx* c, const uep_plan_out& plan, int n_tensors, void* const* main_grad,
                       void* const* slot_grad, const size_t* bytes, cudaStream_t s) {
  RedArgs a;
  a.n_tensors = n_tensors;
  for (int j = 0; j < n_tensors; ++j) {
    a.main_grad[j] = static_cast<float*>(main_grad[j]);
    a.slot_grad[j] = static_cast<float*>(slot_grad[j]);
    a.bytes[j] = bytes[j];
  }
  grad_reduce_kernel<<<2 * c->sm_count, kRedThreads, 0, s>>>(a, c->cfg.E, c->cfg.n_slot, c->M,
                                                           plan.inst_off, plan.inst_rank,
                                                           plan.inst_phys);
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

int launch_inverse(const Ctx* c, const int32_t* out_rank, const int32_t* out_offset,
                   const uep_plan_out& plan, int32_t* out_src, cudaStream_t s) {
  if (c->S == 0) return UEP_OK;
  inverse_kernel<<<(c->S + 255) / 256, 256, 0, s>>>(out_rank, out_offset, plan.rank_base, c->S,
                                                   c->cfg.R, out_src);
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

}  // namespace uep
