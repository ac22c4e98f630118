// uep_internal.cuh — shared declarations of the CUDA path (sm_100a only).
// Nothing here is shared with oracle/ (the CPU oracle is an independent program).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include "uep.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libuep is written for sm_100a (B200) only"
#endif

namespace uep {

constexpr int kWsHeaderBytes = 256 + 4 * UEP_MAX_E;   // from byte 256: acc[E], the histogram's accumulator (zero between calls)
constexpr int kHistThreads = 1024;
constexpr int kRemapThreads = 512;
constexpr int kRemapWarps = kRemapThreads / 32;
constexpr int kRemapItems = 16;          // slots per lane per round (register-resident)
constexpr int kRemapRound = kRemapThreads * kRemapItems;   // 8192 slots per CTA
constexpr int kPlanThreads = 512;       // 16 warps per CTA (8 probe), ~96 registers: a whole SM's register file for two CTAs' worth
constexpr int kPlanLevels = 6;           // bisection levels speculated per round (63 probes over a cluster of 8 CTAs)
constexpr int kPackTile = 16 * 1024;     // bytes per bulk-copy tile
constexpr int kPackStages = 8;           // shared-memory ring depth
constexpr int kMinChunk = 2048;          // smallest histogram/remap chunk (slots per CTA)
constexpr int kMaxChunk = kRemapRound;   // largest: one register-resident round per CTA
constexpr int kPackedEBits = 9;          // packed slot word: expert id | (rank inside chunk << 9); -1 invalid

struct Ctx {
  uep_config cfg;
  int S;                  // T*k
  int M, P;               // main / physical slots per rank
  int E_pad;              // E rounded up to a multiple of 4 (row pitch of the chunk table)
  int n_chunks, chunk_len;        // histogram geometry: one CTA per chunk, one chunk per SM
  int r_chunks, r_chunk_len;      // remap geometry (rank + lookup kernels): <= kMaxChunk slots per CTA
  // source-aware remap (uep_remap_local): chunks never straddle a source rank's block of T/R
  // tokens; l_cpg chunks per source rank, the last one of a block may be shorter.  l_cpg == 0:
  // unsupported shape (T not a multiple of R)
  int l_cpg, l_chunk_len, l_chunks, l_group_len;
  int sm_count;
  int pack_ctas;
  int plan_cluster;       // CTAs per plan solve (thread-block cluster size)
  int prio_high;          // greatest stream priority of the device (launch priority of the planner)
  // static layout, device
  int32_t* d_home;        // [E]   h(e)
  int32_t* d_main_phys;   // [E]   index of e among E_{h(e)} ascending
  int32_t* d_roff;        // [R+1] CSR of E_r
  int32_t* d_rexp;        // [E]   experts grouped by home rank, ascending e
  // work counters of the streaming kernels (pack, grad_reduce): kCtrSlots pairs {next unit,
  // finished CTAs}, zero between launches (the kernels rearm them); launches take the pairs round
  // robin, so up to kCtrSlots such kernels of one context may be in flight at a time
  unsigned* d_ctr;
  unsigned ctr_next;      // host, advanced atomically
  unsigned long long n_launches;   // host, advanced atomically: kernels launched through this context
  // fork/join for uep_balance
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_join, ev_rank;
};

constexpr int kCtrSlots = 64;
unsigned* next_counter(const Ctx* c);     // the next {unit, done} counter pair (thread-safe)
// every launch_* below reports its kernel launches here (uep_launch_count; the bench's gpu_launches)
inline void count_launch(const Ctx* c, int n = 1) {
  __atomic_fetch_add(&const_cast<Ctx*>(c)->n_launches, (unsigned long long)n, __ATOMIC_RELAXED);
}

struct PackArgs {
  const unsigned char* src[UEP_MAX_TENSORS];
  unsigned char* dst[UEP_MAX_TENSORS];
  unsigned long long bytes[UEP_MAX_TENSORS];
  int n_tensors;
};

int set_cuda_error(cudaError_t e);

// An SM's L1 / shared-memory split is chosen for the kernels running on it; a kernel whose shared
// memory does not fit into the current split waits until the SM has drained (measured: rank_kernel
// CTAs, 32 KB, did not start beside hist_kernel CTAs, 33 KB, although registers and threads allowed
// it — the histogram's split was 64 KB).  Every kernel that takes part in uep_balance therefore asks
// for the largest shared-memory carveout; none of them depends on L1 hit rates.
template <typename K>
inline int prefer_max_smem(K kernel) {
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  return e == cudaSuccess ? UEP_OK : set_cuda_error(e);
}

// every CTA adds its counts to ws_acc(ws) with fire-and-forget reductions.  red = true
// (uep_balance): the planner (launch_plan with acc) reads them there and publishes expert_count,
// the lookup zeroes the accumulator again.  red = false: publish_kernel does both.
int launch_histogram(const Ctx* c, const int32_t* ids, int32_t* count, void* ws, cudaStream_t s,
                     bool red = false);
int launch_plan(const Ctx* c, const int32_t* count, const uep_plan_out& plan, cudaStream_t s,
                bool pdl = false, int n_inst = 1, int32_t* acc = nullptr, int32_t* count_out = nullptr,
                int acc_rows = 1, int acc_pitch = 0, int32_t* zero_ptr = nullptr, int zero_n = 0);
// uep_remap = launch_rank (plan-independent: stable rank of every slot inside its chunk, packed
// with the expert id into the workspace) + launch_lookup (plan-dependent: cumulative-quota lookup).
int launch_rank(const Ctx* c, const int32_t* ids, void* ws, cudaStream_t s, bool local = false,
                int chunk0 = 0, int n_launch = -1, bool with_prefix = true, bool bitmaps = true,
                bool write_counts = true);
// token-sharded path: the grouped chunks' count rows alone (hist.cu)
int launch_shard_hist(const Ctx* c, const int32_t* ids, void* ws, cudaStream_t s, int chunk0, int n_launch);
int launch_prefix(const Ctx* c, void* ws, cudaStream_t s, bool local, bool pdl = false);
// token-sharded path: the shard's rows of Lambda[R][E_pad] from its chunks' counts (after the exchange
// the planner sums the matrix's columns and the lookup derives its chunk bases from it: no prefix kernel)
int launch_shard_rows(const Ctx* c, void* ws, cudaStream_t s, int rank0, int n_ranks);
int launch_reroute(const Ctx* c, const uep_plan_out& plan, int32_t* n_inflight, void* ws, cudaStream_t s);
int launch_lookup(const Ctx* c, const void* gate, const uep_plan_out& plan, int32_t* out_replica,
                  int32_t* out_rank, int32_t* out_offset, void* out_gate, void* ws, cudaStream_t s,
                  bool pdl = false, bool local = false, int32_t* n_inflight = nullptr,
                  int32_t* acc_clear = nullptr, int chunk0 = 0, int n_launch = -1, bool src_aware = true,
                  bool from_lambda = false);
int launch_remap(const Ctx* c, const int32_t* ids, const void* gate, const uep_plan_out& plan,
                 int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                 void* ws, cudaStream_t s);
int launch_pack(const Ctx* c, const uep_plan_out& plan, const PackArgs& a, cudaStream_t s);
int launch_grad_reduce(const Ctx* c, const uep_plan_out& plan, int n_tensors, void* const* main_grad,
                       void* const* slot_grad, const size_t* bytes, cudaStream_t s);
int launch_relay(const Ctx* c, const uep_plan_out& plan, int32_t* parent, int32_t* send_volume,
                 cudaStream_t s);
int launch_inverse(const Ctx* c, const int32_t* out_rank, const int32_t* out_offset,
                   const uep_plan_out& plan, int32_t* out_src, cudaStream_t s);
struct Ctx;
int init_plan_kernels(Ctx* c);    // opt-in shared memory attributes, cluster size
int init_remap_kernels();
int init_pack_kernels();
int init_reduce_kernels();

int init_hist_kernels();

#ifdef __CUDACC__
// Programmatic dependent launch (sm_90+).  pdl_trigger: the next kernel in the stream, if it was
// launched with programmatic stream serialization, may start now (its prologue overlaps this
// kernel).  pdl_wait: block until the preceding kernel has completed and its writes are visible;
// a no-op when the kernel was launched normally.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- mbarrier + bulk-copy (TMA engine, 1-D cp.async.bulk) wrappers shared by the streaming kernels
// (pack.cu, reduce.cu) and the histogram's chunk staging (hist.cu) ---------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global, tracked by the thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src_smem)),
               "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
#endif

inline int32_t* ws_table(void* ws) {
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + kWsHeaderBytes);
}
inline int32_t* ws_acc(void* ws) { return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + 256); }
inline size_t ws_table_bytes(const Ctx* c) {
  return (sizeof(int32_t) * (size_t)c->n_chunks * c->E_pad + 255) & ~(size_t)255;
}
inline size_t ws_prefix_bytes(const Ctx* c) {            // [max(r_chunks, l_chunks) + 1][E_pad]
  const size_t rows = (size_t)(c->r_chunks > c->l_chunks ? c->r_chunks : c->l_chunks) + 1;
  return (sizeof(int32_t) * rows * c->E_pad + 255) & ~(size_t)255;
}
inline size_t ws_packed_bytes(const Ctx* c) {
  return sizeof(int32_t) * (((size_t)c->S + 63) & ~(size_t)63);
}
inline size_t ws_reroute_ints(const Ctx* c) {             // cumq and srcpre: [R][E + R*n_slot] each
  return c->l_cpg ? 2 * (size_t)c->cfg.R * (size_t)(c->cfg.E + c->cfg.R * c->cfg.n_slot) : 0;
}
inline int32_t* ws_prefix(const Ctx* c, void* ws) {      // exclusive prefix over remap chunks (+ totals row)
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + kWsHeaderBytes + ws_table_bytes(c));
}
inline int32_t* ws_counts(const Ctx* c, void* ws) {      // per-chunk expert counts, row c = chunk c (never scanned)
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + kWsHeaderBytes + ws_table_bytes(c) +
                                    ws_prefix_bytes(c));
}
inline int32_t* ws_packed(const Ctx* c, void* ws) {      // [S] packed (expert, rank in chunk)
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + kWsHeaderBytes + ws_table_bytes(c) +
                                    2 * ws_prefix_bytes(c));
}
inline int32_t* ws_reroute(const Ctx* c, void* ws) {     // source-aware split tables (uep_remap_local)
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + kWsHeaderBytes + ws_table_bytes(c) +
                                    2 * ws_prefix_bytes(c) + ws_packed_bytes(c));
}
inline size_t ws_lambda_offset(const Ctx* c) {           // Lambda[R][E_pad]: the count matrix of the token-sharded path
  return ((size_t)kWsHeaderBytes + ws_table_bytes(c) + 2 * ws_prefix_bytes(c) + ws_packed_bytes(c) +
          sizeof(int32_t) * ws_reroute_ints(c) + 255) & ~(size_t)255;
}
inline size_t ws_lambda_bytes(const Ctx* c) { return c->l_cpg ? sizeof(int32_t) * (size_t)c->cfg.R * c->E_pad : 0; }
inline int32_t* ws_lambda(const Ctx* c, void* ws) {
  return reinterpret_cast<int32_t*>(static_cast<unsigned char*>(ws) + ws_lambda_offset(c));
}

}  // namespace uep

#define UEP_CUDA_TRY(expr)                                   \
  do {                                                       \
    cudaError_t _e = (expr);                                 \
    if (_e != cudaSuccess) return ::uep::set_cuda_error(_e); \
  } while (0)
