// relay.cu — uep_relay_plan: load-aware relay scheduling, topology only (
// §6.2 "Chunk Streaming Relay for Hotspot Fan-Out").
//
// For every expert with more than 4 replicas a two-stage tree replaces the source's direct
// fan-out: k = sqrt(f) (to nearest) first-stage relays chosen among the expert's replica ranks
// with the smallest sending volume, every other replica attached to the relay whose volume would
// remain smallest after taking it; volumes are updated before the next hot expert.  The transfers
// themselves (chunk streaming between GPUs) are out of scope; this kernel only decides the trees.
// A few hot experts, a few dozen replicas each: one warp, arg-min by redux.sync.min on a packed
// key (volume << 8 | rank id gives "smallest volume, lowest rank id" in one instruction).
#include "uep_internal.cuh"

namespace uep {

constexpr unsigned kRelayFull = 0xffffffffu;
constexpr int kRelayThreshold = 4;
constexpr int kRelayPerLane = UEP_MAX_R / 32; // replicas of one expert per lane

__device__ __forceinline__ int relay_frontier(int f) {      // sqrt(f) to nearest, in integers
  int k = (int)sqrtf((float)f);
  while (k * k > f) --k;
  while ((k + 1) * (k + 1) <= f) ++k;
  return (f > k * k + k) ? k + 1 : k;
}

__global__ void __launch_bounds__(32)
relay_kernel(int E, int R, int cap, const int32_t* __restrict__ inst_off,
             const int32_t* __restrict__ inst_rank, const int32_t* __restrict__ home,
             int32_t* __restrict__ parent, int32_t* __restrict__ send_volume) {
  __shared__ int vol[UEP_MAX_R];
  __shared__ int is_relay[UEP_MAX_R];
  const int lane = threadIdx.x;
  for (int r = lane; r < R; r += 32) { vol[r] = 0; is_relay[r] = 0; }
  for (int p = lane; p < cap; p += 32) parent[p] = -1;
  __syncwarp();
  // 1. direct sends: every replica hangs off its expert's home rank
  for (int e = lane; e < E; e += 32) {
    const int lo = inst_off[e], hi = inst_off[e + 1], h = home[e];
    if (hi - lo > 1) atomicAdd(&vol[h], hi - lo - 1);
    for (int p = lo + 1; p < hi; ++p) parent[p] = h;
  }
  __syncwarp();
  // 2. relay-eligible experts one by one, ascending expert id (S24)
  for (int e = 0; e < E; ++e) {
    const int lo = inst_off[e], f = inst_off[e + 1] - lo - 1;
    if (f <= kRelayThreshold) continue;
    const int k = relay_frontier(f), h = home[e];
    int rk[kRelayPerLane];                       // ranks of this lane's replicas (i = lane + 32 q)
    unsigned chosen = 0;
#pragma unroll
    for (int q = 0; q < kRelayPerLane; ++q) {
      const int i = lane + 32 * q;
      rk[q] = (i < f) ? inst_rank[lo + 1 + i] : -1;
    }
    // 3. k relays: smallest sending volume, ties -> lower rank id.  Lane j keeps relay j.
    int my_relay = -1, my_leaves = 0;
    for (int j = 0; j < k; ++j) {
      unsigned key = 0xffffffffu;
#pragma unroll
      for (int q = 0; q < kRelayPerLane; ++q)
        if (rk[q] >= 0 && !((chosen >> q) & 1u)) key = min(key, ((unsigned)vol[rk[q]] << 8) | (unsigned)rk[q]);
      const unsigned best = __reduce_min_sync(kRelayFull, key);
      const int w = (int)(best & 255u);
#pragma unroll
      for (int q = 0; q < kRelayPerLane; ++q)
        if (rk[q] == w) { chosen |= 1u << q; is_relay[w] = 1; }
      if (lane == j) my_relay = w;
    }
    __syncwarp();
    // 4. leaves in instance order: the relay whose volume would remain smallest after taking it
    for (int i = 0; i < f; ++i) {
      const int r = inst_rank[lo + 1 + i];
      if (is_relay[r]) continue;
      const unsigned key = (my_relay >= 0) ? (((unsigned)(vol[my_relay] + my_leaves + 1) << 8) | (unsigned)my_relay)
                                           : 0xffffffffu;
      const unsigned best = __reduce_min_sync(kRelayFull, key);
      const int b = (int)(best & 255u);
      if (my_relay == b) my_leaves += 1;
      if (lane == 0) parent[lo + 1 + i] = b;
    }
    __syncwarp();
    // 5. the source now sends k copies instead of f, each relay its leaves
    if (lane == 0) vol[h] += k - f;
    __syncwarp();
    if (my_relay >= 0) { vol[my_relay] += my_leaves; is_relay[my_relay] = 0; }
    __syncwarp();
  }
  for (int r = lane; r < R; r += 32) send_volume[r] = vol[r];
}

int launch_relay(const Ctx* c, const uep_plan_out& plan, int32_t* parent, int32_t* send_volume,
                 cudaStream_t s) {
  relay_kernel<<<1, 32, 0, s>>>(c->cfg.E, c->cfg.R, c->cfg.E + c->cfg.R * c->cfg.n_slot, plan.inst_off,
                                plan.inst_rank, c->d_home, parent, send_volume);
  UEP_CUDA_TRY(cudaGetLastError());
  count_launch(c);
  return UEP_OK;
}

}  // namespace uep
