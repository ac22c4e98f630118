// pack.cu — uep_pack: forward weight distribution main -> redundant slot (§4.2),
// single-GPU part: copy the state of every replicated expert into the destination
// rank's slot buffer.  dst[j][(t*n_slot+s)*B_j ..) = src[j][e*B_j ..) for x_{t,s} = e.
//
// HBM-bound byte movement.  Kept from the paper's tile streaming (§6.1): fixed
// tiles, a persistent grid, and "each source tile is staged once into shared memory and stored
// to all replica destinations" — so an expert with f replicas costs 1 read + f writes.
// B200 form: the staging is done by the TMA engine, not by threads.  One elected thread per
// CTA drives a ring of kPackStages shared-memory tiles: cp.async.bulk global->shared
// (complete_tx on an mbarrier), then one cp.async.bulk shared->global per destination,
// committed as a bulk group; a stage is refilled once the group that read it has drained
// (cp.async.bulk.wait_group.read).  The grid is static and persistent (graph-capturable); the
// work list is read from the plan on the device and handed out in batches from a self-resetting
// counter (see pack_kernel).
#include "uep_internal.cuh"

namespace uep {

constexpr int kPackThreads = 32;
constexpr int kPackPending = 1;          // store groups allowed in flight when a stage is reused
constexpr int kPackAhead = kPackStages - 1 - kPackPending;   // loads issued ahead of the stores

// A unit = one source tile and its destinations.  Units are numbered expert-major over the
// replicated experts only: u = (index of e among replicated experts) * TPE + (tile index over the
// expert's tensors in order), TPE = sum_j ceil(B_j / kPackTile).
struct Unit {
  const unsigned char* src;
  unsigned long long dst_off;   // byte offset of the tile inside a slot of tensor j
  uint32_t bytes;
  int e, j;
};

constexpr unsigned kPackBatch = 8;       // units taken from the shared counter at a time (128 KB)

// Work distribution is DYNAMIC: CTAs take batches of kPackBatch consecutive units from a counter
// in global memory (ctr[0]; the next batch is requested while the current one is being
// processed, so the L2 round trip is hidden).  With a static equal split the kernel ran at the
// pace of its slowest SM: SMs do not all see the same bandwidth (148 streaming CTAs: 0.89 of the
// copy peak; the same static split on 128: 0.97; and 0.86 again when the CTAs landed unevenly
// behind a still-running lookup_kernel).  The last CTA to finish resets the counters (ctr[1]
// counts finished CTAs), so the launch stays graph-replayable.
__global__ void __launch_bounds__(kPackThreads, 1)
pack_kernel(PackArgs a, int E, int n_slot, int M, const int32_t* __restrict__ inst_off,
            const int32_t* __restrict__ inst_rank, const int32_t* __restrict__ inst_phys,
            unsigned* __restrict__ ctr) {
  extern __shared__ __align__(128) unsigned char pack_smem[];
  __shared__ __align__(8) uint64_t full[kPackStages];
  __shared__ Unit ring[kPackStages];
  __shared__ short rexp[UEP_MAX_E];                     // replicated experts, ascending
  const int lane = threadIdx.x;
  int n_rexp = 0;
  for (int base = 0; base < E; base += 32) {            // warp-cooperative compaction
    const int e = base + lane;
    const bool r = e < E && __ldg(inst_off + e + 1) - __ldg(inst_off + e) > 1;
    const unsigned m = __ballot_sync(0xffffffffu, r);
    if (r) rexp[n_rexp + __popc(m & ((1u << lane) - 1u))] = (short)e;
    n_rexp += __popc(m);
  }
  __syncwarp();
  if (lane != 0) return;                                // one elected thread drives the TMA engine
  for (int s = 0; s < kPackStages; ++s) mbar_init(&full[s], 1);
  mbar_fence_init();
  fence_proxy_async();

  unsigned tiles_of[UEP_MAX_TENSORS];
  unsigned tpe = 0;
#pragma unroll
  for (int j = 0; j < UEP_MAX_TENSORS; ++j) {
    tiles_of[j] = j < a.n_tensors ? (unsigned)((a.bytes[j] + kPackTile - 1) / kPackTile) : 0u;
    tpe += tiles_of[j];
  }
  const unsigned total = (unsigned)n_rexp * tpe;        // < 2^31: checked by launch_pack

  // batch state: units [cur, cur_end) decoded incrementally as (ri, j, tile)
  unsigned cur = 0, cur_end = 0, ri = 0, tile = 0;
  int j = 0;
  unsigned nxt = atomicAdd(ctr, kPackBatch);            // first batch
  bool more = true;
  auto next = [&](Unit& u) -> bool {
    if (cur == cur_end) {
      if (nxt >= total) return false;
      cur = nxt;
      cur_end = min(nxt + kPackBatch, total);
      nxt = atomicAdd(ctr, kPackBatch);                 // requested now, needed a batch later
      ri = cur / tpe;
      unsigned r = cur - ri * tpe;
      j = 0;
      while (r >= tiles_of[j]) { r -= tiles_of[j]; ++j; }
      tile = r;
    }
    const unsigned long long B = a.bytes[j];
    const unsigned long long off = (unsigned long long)tile * kPackTile;
    u.e = rexp[ri]; u.j = j;
    u.src = a.src[j] + (unsigned long long)u.e * B + off;
    u.dst_off = off;
    u.bytes = (uint32_t)min((unsigned long long)kPackTile, B - off);
    ++cur;
    if (++tile == tiles_of[j]) {
      tile = 0;
      do { ++j; } while (j < a.n_tensors && tiles_of[j] == 0);
      if (j >= a.n_tensors) {
        ++ri;
        j = 0;
        while (j < a.n_tensors && tiles_of[j] == 0) ++j;
      }
    }
    return true;
  };

  long long n_loaded = 0, n_stored = 0;
  auto issue_load = [&]() {
    Unit u;
    if (!more || !(more = next(u))) return;
    const int st = (int)(n_loaded % kPackStages);
    ring[st] = u;
    mbar_expect_tx(&full[st], u.bytes);
    bulk_g2s(pack_smem + (size_t)st * kPackTile, u.src, u.bytes, &full[st]);
    ++n_loaded;
  };
  for (int i = 0; i < kPackAhead; ++i) issue_load();
  while (n_stored < n_loaded) {
    // refill: the stage to be overwritten was read by the store group of unit n_loaded-kPackStages,
    // which is at least kPackPending+1 groups old
    if (more) {
      if (n_loaded >= kPackStages) bulk_wait_read<kPackPending>();
      issue_load();
    }
    const int st = (int)(n_stored % kPackStages);
    mbar_wait(&full[st], (uint32_t)((n_stored / kPackStages) & 1));
    fence_proxy_async();
    const Unit u = ring[st];
    const int lo = inst_off[u.e], hi = inst_off[u.e + 1];
    const unsigned long long B = a.bytes[u.j];
    for (int p = lo + 1; p < hi; ++p) {                  // every replica of e (entry lo = main)
      const int slot = inst_rank[p] * n_slot + (inst_phys[p] - M);
      bulk_s2g(a.dst[u.j] + (unsigned long long)slot * B + u.dst_off,
               pack_smem + (size_t)st * kPackTile, u.bytes);
    }
    bulk_commit();
    ++n_stored;
  }
  // every request of this CTA has returned; the last CTA to get here rearms the counters
  __threadfence();
  if (atomicAdd(ctr + 1, 1u) == gridDim.x - 1) {
    ctr[0] = 0u;
    ctr[1] = 0u;
    __threadfence();
  }
  bulk_wait_all();
}

int init_pack_kernels() {
  if (prefer_max_smem(pack_kernel) != UEP_OK) return UEP_ERR_CUDA;
  UEP_CUDA_TRY(cudaFuncSetAttribute(pack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kPackStages * kPackTile));
  return UEP_OK;
}

int launch_pack(const Ctx* c, const uep_plan_out& plan, const PackArgs& a, cudaStream_t s) {
  unsigned long long tpe = 0;
  for (int j = 0; j < a.n_tensors; ++j) tpe += (a.bytes[j] + kPackTile - 1) / kPackTile;
  if (tpe * (unsigned long long)c->cfg.E >= (1ull << 31) - (unsigned long long)kPackBatch * 4096) return UEP_ERR_UNSUPPORTED;
  pack_kernel<<<c->pack_ctas, kPackThreads, kPackStages * kPackTile, s>>>(
      a, c->cfg.E, c->cfg.n_slot, c->M, plan.inst_off, plan.inst_rank, plan.inst_phys, next_counter(c));
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

}  // namespace uep
