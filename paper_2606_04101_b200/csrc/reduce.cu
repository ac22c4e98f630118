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
// writes (1+f) B (the sum, and zeros).  Kept from the paper: fixed tiles, a persistent grid
// (capturable although the work list is data-dependent), shared-memory tiles filled ahead of the
// reduction.  B200 form: one elected producer thread per CTA streams 8 KB tiles (main, then each
// replica, in instance order) into a 16-stage shared-memory ring with cp.async.bulk on mbarriers;
// four consumer warps add them in that order (so the fp32 result is bit-identical run to run and
// equal to a sequential fp32 sum), release each stage as soon as they have read it, and one of
// them sends the reduced tile and the zero tiles back with cp.async.bulk shared->global.  A first
// version with register-resident loads (no ring) reached 0.23-0.29 of the HBM peak: one batch of
// loads in flight per thread is not enough memory parallelism; the ring with a static split of
// the tiles reached 0.90, with the dynamic hand-out below 0.97+.
#include "uep_internal.cuh"

namespace uep {

constexpr int kRedConsumers = 128;                           // 4 consumer warps; warp 0 is the producer
constexpr int kRedThreads = 32 + kRedConsumers;
constexpr int kRedTile = 8 * 1024;                           // bytes per tile = 128 threads x 4 float4
constexpr int kRedVec = kRedTile / 16 / kRedConsumers;       // float4 per consumer thread per tile
constexpr int kRedStages = 16;                               // shared-memory ring of load tiles (128 KB)

struct RedArgs {
  float* main_grad[UEP_MAX_TENSORS];
  float* slot_grad[UEP_MAX_TENSORS];
  unsigned long long bytes[UEP_MAX_TENSORS];
  int n_tensors;
};

// A unit = one tile of the main buffer and the same tile of every replica slot: 1 + f ring
// stages.  Units are numbered expert-major over the replicated experts (as in pack.cu) and handed
// out DYNAMICALLY in batches of kRedBatch from a self-resetting counter in global memory (a
// static equal split runs at the pace of the slowest SM: 0.90 of the copy peak instead of 0.97+).
// The producer takes the batches and tells the consumers what each unit is through a small ring
// of descriptors in shared memory, published before the unit's first stage is armed.
struct RedUnit {
  unsigned long long off;       // byte offset of the tile inside tensor j of an expert / slot
  int e, j, lo, f;              // f < 0: no more work
  uint32_t bytes;
  int pad;
};
constexpr unsigned kRedBatch = 8;
constexpr int kRedUnitRing = kRedStages;     // >= 2 stages per unit: at most kRedStages/2 units in flight

__global__ void __launch_bounds__(kRedThreads, 1)
grad_reduce_kernel(RedArgs a, int E, int n_slot, int M, const int32_t* __restrict__ inst_off,
                   const int32_t* __restrict__ inst_rank, const int32_t* __restrict__ inst_phys,
                   unsigned* __restrict__ ctr) {
  extern __shared__ __align__(128) unsigned char red_smem[];
  unsigned char* ring = red_smem;                                    // [kRedStages][kRedTile]
  unsigned char* outbuf = ring + (size_t)kRedStages * kRedTile;      // [2][kRedTile] reduced main tiles
  unsigned char* zero = outbuf + 2 * kRedTile;                       // [kRedTile] zeros
  __shared__ __align__(8) uint64_t full[kRedStages], empty[kRedStages];
  __shared__ __align__(16) RedUnit units[kRedUnitRing];
  __shared__ short rexp[UEP_MAX_E];                                  // replicated experts, ascending
  const int tid = threadIdx.x;
  for (int i = tid; i < kRedTile / 16; i += kRedThreads)
    reinterpret_cast<float4*>(zero)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (tid == 0) {
    for (int s = 0; s < kRedStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kRedConsumers); }
    mbar_fence_init();
  }
  fence_proxy_async();                                               // zero tile visible to bulk stores
  __syncthreads();
  auto slot_of = [&](int p) { return __ldg(inst_rank + p) * n_slot + (__ldg(inst_phys + p) - M); };

  if (tid < 32) {
    // ---- producer warp: compact the replicated experts, then one elected thread streams tiles --
    int n_rexp = 0;
    for (int base = 0; base < E; base += 32) {
      const int e = base + tid;
      const bool r = e < E && __ldg(inst_off + e + 1) - __ldg(inst_off + e) > 1;
      const unsigned m = __ballot_sync(0xffffffffu, r);
      if (r) rexp[n_rexp + __popc(m & ((1u << tid) - 1u))] = (short)e;
      n_rexp += __popc(m);
    }
    __syncwarp();
    if (tid != 0) return;
    unsigned tiles_of[UEP_MAX_TENSORS];
    unsigned tpe = 0;
#pragma unroll
    for (int j = 0; j < UEP_MAX_TENSORS; ++j) {
      tiles_of[j] = j < a.n_tensors ? (unsigned)((a.bytes[j] + kRedTile - 1) / kRedTile) : 0u;
      tpe += tiles_of[j];
    }
    const unsigned total = (unsigned)n_rexp * tpe;                   // < 2^31: checked at launch
    unsigned long long n = 0, unit = 0;                              // ring position, unit counter
    auto acquire = [&]() {                                           // stage n % kRedStages is free again
      const int st = (int)(n % kRedStages);
      if (n >= kRedStages) mbar_wait(&empty[st], (uint32_t)(((n / kRedStages) - 1) & 1));
      return st;
    };
    auto load = [&](const unsigned char* src, uint32_t bytes) {
      const int st = acquire();
      mbar_expect_tx(&full[st], bytes);
      bulk_g2s(ring + (size_t)st * kRedTile, src, bytes, &full[st]);
      ++n;
    };
    unsigned nxt = atomicAdd(ctr, kRedBatch);
    while (nxt < total) {
      const unsigned cur0 = nxt, cur_end = min(nxt + kRedBatch, total);
      nxt = atomicAdd(ctr, kRedBatch);                               // requested now, needed a batch later
      unsigned ri = cur0 / tpe, r = cur0 - ri * tpe;
      int j = 0;
      while (r >= tiles_of[j]) { r -= tiles_of[j]; ++j; }
      unsigned tile = r;
      for (unsigned u = cur0; u < cur_end; ++u) {
        const int e = rexp[ri];
        const int lo = __ldg(inst_off + e), f = __ldg(inst_off + e + 1) - lo - 1;
        const unsigned long long B = a.bytes[j], off = (unsigned long long)tile * kRedTile;
        const uint32_t bytes = (uint32_t)min((unsigned long long)kRedTile, B - off);
        acquire();                                                   // before the descriptor slot is rewritten
        RedUnit& d = units[unit % kRedUnitRing];
        d.off = off; d.e = e; d.j = j; d.lo = lo; d.f = f; d.bytes = bytes;
        load(reinterpret_cast<const unsigned char*>(a.main_grad[j]) + (unsigned long long)e * B + off, bytes);
        for (int q = 1; q <= f; ++q)
          load(reinterpret_cast<const unsigned char*>(a.slot_grad[j]) + (unsigned long long)slot_of(lo + q) * B + off, bytes);
        ++unit;
        if (++tile == tiles_of[j]) {
          tile = 0;
          do { ++j; } while (j < a.n_tensors && tiles_of[j] == 0);
          if (j >= a.n_tensors) {
            ++ri;
            j = 0;
            while (j < a.n_tensors && tiles_of[j] == 0) ++j;
          }
        }
      }
    }
    {                                                                // end marker: an empty stage
      const int st = acquire();
      units[unit % kRedUnitRing].f = -1;
      mbar_arrive(&full[st]);
    }
    __threadfence();                                                 // every request has returned
    if (atomicAdd(ctr + 1, 1u) == gridDim.x - 1) {                   // last CTA rearms the counters
      ctr[0] = 0u;
      ctr[1] = 0u;
      __threadfence();
    }
    return;
  }

  // ---- consumers: 128 threads, 4 float4 each per tile --------------------------------------------
  const int ct = tid - 32;
  unsigned long long n = 0, unit = 0;
  while (true) {
    {                                                    // the unit's first stage also publishes its descriptor
      const int st = (int)(n % kRedStages);
      mbar_wait(&full[st], (uint32_t)((n / kRedStages) & 1));
    }
    const RedUnit d = units[unit % kRedUnitRing];
    if (d.f < 0) break;
    const int e = d.e, j = d.j, lo = d.lo, f = d.f;
    const unsigned long long off = d.off;
    const uint32_t bytes = d.bytes;
    const int n4 = (int)(bytes >> 4);
    float4 acc[kRedVec];
    for (int q = 0; q <= f; ++q) {                       // instance order: main, replica 1, 2, ...
      const int st = (int)(n % kRedStages);
      if (q) mbar_wait(&full[st], (uint32_t)((n / kRedStages) & 1));
      const float4* t = reinterpret_cast<const float4*>(ring + (size_t)st * kRedTile);
#pragma unroll
      for (int v = 0; v < kRedVec; ++v) {
        const int i = v * kRedConsumers + ct;
        const float4 x = (i < n4) ? t[i] : make_float4(0.f, 0.f, 0.f, 0.f);
        if (q == 0) acc[v] = x;
        else { acc[v].x += x.x; acc[v].y += x.y; acc[v].z += x.z; acc[v].w += x.w; }
      }
      mbar_arrive(&empty[st]);                       // this thread is done with the stage
      ++n;
    }
    // (A) the elected thread has waited until the stores of unit-2 finished reading outbuf[unit&1]
    asm volatile("bar.sync 1, %0;" ::"n"(kRedConsumers) : "memory");
    float4* ob = reinterpret_cast<float4*>(outbuf + (size_t)(unit & 1) * kRedTile);
#pragma unroll
    for (int v = 0; v < kRedVec; ++v) {
      const int i = v * kRedConsumers + ct;
      if (i < n4) ob[i] = acc[v];
    }
    fence_proxy_async();
    asm volatile("bar.sync 1, %0;" ::"n"(kRedConsumers) : "memory");      // (B) tile complete in shared memory
    if (ct == 0) {
      const unsigned long long B = a.bytes[j];
      bulk_s2g(reinterpret_cast<unsigned char*>(a.main_grad[j]) + (unsigned long long)e * B + off, ob, bytes);
      for (int q = 1; q <= f; ++q)                       // cleared in place
        bulk_s2g(reinterpret_cast<unsigned char*>(a.slot_grad[j]) + (unsigned long long)slot_of(lo + q) * B + off,
                     zero, bytes);
      bulk_commit();
      bulk_wait_read<1>();                               // unit-1's stores have read their smem
    }
    ++unit;
  }
  if (ct == 0) bulk_wait_all();
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

int init_reduce_kernels() {
  UEP_CUDA_TRY(cudaFuncSetAttribute(grad_reduce_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (kRedStages + 3) * kRedTile));
  return UEP_OK;
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
  const size_t smem = (size_t)(kRedStages + 3) * kRedTile;
  unsigned long long tpe = 0;
  for (int j = 0; j < n_tensors; ++j) tpe += (bytes[j] + kRedTile - 1) / kRedTile;
  if (tpe * (unsigned long long)c->cfg.E >= (1ull << 31) - (unsigned long long)kRedBatch * 4096) return UEP_ERR_UNSUPPORTED;
  grad_reduce_kernel<<<c->pack_ctas, kRedThreads, smem, s>>>(a, c->cfg.E, c->cfg.n_slot, c->M,
                                                            plan.inst_off, plan.inst_rank,
                                                            plan.inst_phys, next_counter(c));
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

int launch_inverse(const Ctx* c, const int32_t* out_rank, const int32_t* out_offset,
                   const uep_plan_out& plan, int32_t* out_src, cudaStream_t s) {
  if (c->S == 0) return UEP_OK;
  inverse_kernel<<<(c->S + 255) / 256, 256, 0, s>>>(out_rank, out_offset, plan.rank_base, c->S,
                                                   c->cfg.R, out_src);
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

}  // namespace uep
