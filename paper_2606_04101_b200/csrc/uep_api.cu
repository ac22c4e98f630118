// uep_api.cu — C-ABI entry points: context, argument checks, stage chaining (include/uep.h).
// Host logic only; every step of the path runs in the kernels of hist.cu / plan.cu /
// remap.cu / pack.cu.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#include <algorithm>
#include "uep_internal.cuh"

namespace uep {

static thread_local char g_cuda_err[256] = "";

int set_cuda_error(cudaError_t e) {
  std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", cudaGetErrorName(e),
                cudaGetErrorString(e));
  return UEP_ERR_CUDA;
}

unsigned* next_counter(const Ctx* c) {
  Ctx* m = const_cast<Ctx*>(c);                // the round-robin index is the context's only mutable state
  const unsigned i = __atomic_fetch_add(&m->ctr_next, 1u, __ATOMIC_RELAXED);
  return m->d_ctr + 2 * (i % kCtrSlots);
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static int check_plan_ptrs(const Ctx* c, const uep_plan_out* p) {
  if (!p) return UEP_ERR_INVALID_ARG;
  const void* req[] = {p->slot_expert, p->inst_off,  p->inst_rank, p->inst_phys, p->inst_cum, p->inst_base,
                       p->phys_count,  p->phys_base, p->rank_load, p->rank_base, p->scalars};
  for (const void* q : req)
    if (!q || !aligned16(q)) return UEP_ERR_INVALID_ARG;
  if (p->U && !aligned16(p->U)) return UEP_ERR_INVALID_ARG;
  (void)c;
  return UEP_OK;
}

static int fill_pack_args(int32_t n_tensors, const void* const* src, const size_t* bytes,
                          void* const* dst, PackArgs& a) {
  if (n_tensors < 0 || n_tensors > UEP_MAX_TENSORS) return UEP_ERR_INVALID_ARG;
  a.n_tensors = n_tensors;
  if (n_tensors && (!src || !bytes || !dst)) return UEP_ERR_INVALID_ARG;
  for (int j = 0; j < n_tensors; ++j) {
    if (!src[j] || !dst[j] || !aligned16(src[j]) || !aligned16(dst[j])) return UEP_ERR_INVALID_ARG;
    if (bytes[j] == 0 || (bytes[j] & 15)) return UEP_ERR_INVALID_ARG;
    a.src[j] = static_cast<const unsigned char*>(src[j]);
    a.dst[j] = static_cast<unsigned char*>(dst[j]);
    a.bytes[j] = bytes[j];
  }
  return UEP_OK;
}

}  // namespace uep

using namespace uep;

extern "C" {

int uep_create(const uep_config* cfg, uep_ctx** out) {
  if (!cfg || !out) return UEP_ERR_INVALID_ARG;
  *out = nullptr;
  if (cfg->T < 0 || cfg->k < 1 || cfg->E < 1 || cfg->R < 1 || cfg->n_slot < 0 ||
      cfg->u_min < 1 || cfg->beta_num < 1 || cfg->beta_den < 1)
    return UEP_ERR_INVALID_ARG;
  if (cfg->floor_mode != UEP_FLOOR_STRICT && cfg->floor_mode != UEP_FLOOR_TOLERANT)
    return UEP_ERR_INVALID_ARG;
  if (cfg->gate_dtype < UEP_GATE_F32 || cfg->gate_dtype > UEP_GATE_NONE) return UEP_ERR_INVALID_ARG;
  if (cfg->E > UEP_MAX_E || cfg->R > UEP_MAX_R || cfg->n_slot > UEP_MAX_NSLOT)
    return UEP_ERR_UNSUPPORTED;
  const long long S = (long long)cfg->T * cfg->k;
  if (S >= (1LL << 24)) return UEP_ERR_UNSUPPORTED;      // planner packs slack into 24 bits
  if ((long long)cfg->beta_num * ((S + cfg->R - 1) / cfg->R) >= (1LL << 62)) return UEP_ERR_UNSUPPORTED;

  int dev = 0, n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) { cudaGetLastError(); return UEP_ERR_NO_DEVICE; }
  UEP_CUDA_TRY(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  UEP_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major < 10) return UEP_ERR_UNSUPPORTED;       // sm_100a only

  Ctx* c = new (std::nothrow) Ctx();
  if (!c) return UEP_ERR_INVALID_ARG;
  std::memset(c, 0, sizeof(Ctx));
  c->cfg = *cfg;
  c->cfg.home_rank = nullptr;                            // never retained
  c->S = (int)S;
  c->sm_count = prop.multiProcessorCount;
  const int E = cfg->E, R = cfg->R;
  c->E_pad = (E + 3) & ~3;

  // static layout (Table 1): h(e), E_r, main slot index
  std::vector<int32_t> home(E), main_phys(E), roff(R + 1, 0), rexp(E);
  for (int e = 0; e < E; ++e) {
    int h = cfg->home_rank ? cfg->home_rank[e] : (int)(((long long)e * R) / E);
    if (h < 0 || h >= R) { delete c; return UEP_ERR_INVALID_ARG; }
    home[e] = h;
    roff[h + 1] += 1;
  }
  int M = 0;
  for (int r = 0; r < R; ++r) { M = std::max(M, roff[r + 1]); roff[r + 1] += roff[r]; }
  {
    std::vector<int32_t> fill(R, 0);
    for (int e = 0; e < E; ++e) {
      main_phys[e] = fill[home[e]];
      rexp[roff[home[e]] + fill[home[e]]] = e;
      fill[home[e]] += 1;
    }
  }
  c->M = M;
  c->P = M + cfg->n_slot;

  // launch geometry.  Histogram: one CTA per chunk, one chunk per SM (whole 128-slot lines).
  // Remap (rank + lookup kernels): chunks of whole 512-slot steps, <= kMaxChunk slots (one
  // register-resident round), about two chunks per SM so that co-resident CTAs overlap their
  // load / rank / store phases.  (Measured: 274 chunks of 7680 slots, so that every lookup CTA is
  // resident beside the planner's 8 SMs, gives a chain of 32.8 us against 32.0 us with 293 x 7168.)
  {
    long long per = (S + c->sm_count - 1) / c->sm_count;
    per = std::max<long long>(per, kMinChunk);
    per = (per + 127) / 128 * 128;
    c->chunk_len = (int)per;
    c->n_chunks = (int)std::max<long long>(1, (S + per - 1) / per);
    const int r_sms = std::max(1, c->sm_count);
    long long rper = (S + 2 * r_sms - 1) / (2 * r_sms);
    rper = std::max<long long>(rper, kMinChunk);
    rper = (rper + kRemapThreads - 1) / kRemapThreads * kRemapThreads;
    rper = std::min<long long>(rper, kMaxChunk);
    c->r_chunk_len = (int)rper;
    c->r_chunks = (int)std::max<long long>(1, (S + rper - 1) / rper);
    // source-aware geometry: every source rank's block of (T/R)*k slots is cut into l_cpg chunks
    c->l_cpg = c->l_chunk_len = c->l_chunks = c->l_group_len = 0;
    if (cfg->T > 0 && cfg->T % R == 0) {
      const long long block = (long long)(cfg->T / R) * cfg->k;
      const long long cpg = (block + kMaxChunk - 1) / kMaxChunk;
      long long len = (block + cpg - 1) / cpg;
      len = std::min<long long>((len + 31) / 32 * 32, kMaxChunk);
      c->l_cpg = (int)cpg;
      c->l_chunk_len = (int)len;
      c->l_chunks = (int)(cpg * R);
      c->l_group_len = (int)block;
    }
  }
  // pack / grad_reduce grid: one persistent streaming CTA per SM; the tiles are handed out
  // dynamically (profiles/r01_pack_grid.md: a static split is bound by the slowest SM)
  c->pack_ctas = c->sm_count;

  auto fail = [&](int rc) { uep_destroy(reinterpret_cast<uep_ctx*>(c)); return rc; };
  cudaError_t e;
#define UEP_TRY_OR_FAIL(x) do { e = (x); if (e != cudaSuccess) return fail(set_cuda_error(e)); } while (0)
  UEP_TRY_OR_FAIL(cudaMalloc(&c->d_home, sizeof(int32_t) * E));
  UEP_TRY_OR_FAIL(cudaMalloc(&c->d_main_phys, sizeof(int32_t) * E));
  UEP_TRY_OR_FAIL(cudaMalloc(&c->d_roff, sizeof(int32_t) * (R + 1)));
  UEP_TRY_OR_FAIL(cudaMalloc(&c->d_rexp, sizeof(int32_t) * E));
  UEP_TRY_OR_FAIL(cudaMalloc(&c->d_ctr, sizeof(unsigned) * 2 * kCtrSlots));
  UEP_TRY_OR_FAIL(cudaMemset(c->d_ctr, 0, sizeof(unsigned) * 2 * kCtrSlots));
  UEP_TRY_OR_FAIL(cudaMemcpy(c->d_home, home.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  UEP_TRY_OR_FAIL(cudaMemcpy(c->d_main_phys, main_phys.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  UEP_TRY_OR_FAIL(cudaMemcpy(c->d_roff, roff.data(), sizeof(int32_t) * (R + 1), cudaMemcpyHostToDevice));
  UEP_TRY_OR_FAIL(cudaMemcpy(c->d_rexp, rexp.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  {
    int least = 0, greatest = 0;
    UEP_TRY_OR_FAIL(cudaDeviceGetStreamPriorityRange(&least, &greatest));
    c->prio_high = greatest;
    // side stream (rank + prefix, pack) at the lowest priority: the critical path runs on the caller's stream
    UEP_TRY_OR_FAIL(cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, least));
  }
  UEP_TRY_OR_FAIL(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
  UEP_TRY_OR_FAIL(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
  UEP_TRY_OR_FAIL(cudaEventCreateWithFlags(&c->ev_rank, cudaEventDisableTiming));
#undef UEP_TRY_OR_FAIL
  int rc = init_plan_kernels(c);
  if (rc == UEP_OK) rc = init_hist_kernels();
  if (rc == UEP_OK) rc = init_remap_kernels();
  if (rc == UEP_OK) rc = init_pack_kernels();
  if (rc == UEP_OK) rc = init_reduce_kernels();
  if (rc != UEP_OK) return fail(rc);
  *out = reinterpret_cast<uep_ctx*>(c);
  return UEP_OK;
}

void uep_destroy(uep_ctx* ctx) {
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (!c) return;
  if (c->d_home) cudaFree(c->d_home);
  if (c->d_main_phys) cudaFree(c->d_main_phys);
  if (c->d_roff) cudaFree(c->d_roff);
  if (c->d_rexp) cudaFree(c->d_rexp);
  if (c->d_ctr) cudaFree(c->d_ctr);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->ev_rank) cudaEventDestroy(c->ev_rank);
  delete c;
}

size_t uep_workspace_bytes(const uep_ctx* ctx) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return 0;
  return ws_lambda_offset(c) + ws_lambda_bytes(c);
}

int uep_workspace_init(const uep_ctx* ctx, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  // the accumulator, and row 0 of the remap prefix table (it stays zero: the scan starts at row 1)
  UEP_CUDA_TRY(cudaMemsetAsync(ws, 0, kWsHeaderBytes, static_cast<cudaStream_t>(stream)));
  UEP_CUDA_TRY(cudaMemsetAsync(ws_prefix(c, ws), 0, ws_prefix_bytes(c), static_cast<cudaStream_t>(stream)));
  return UEP_OK;
}

int uep_plan_bytes(const uep_ctx* ctx, uep_plan_sizes* out) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !out) return UEP_ERR_INVALID_ARG;
  const int E = c->cfg.E, R = c->cfg.R, ns = c->cfg.n_slot;
  out->slot_expert = std::max(1, R * ns);
  out->inst_off = E + 1;
  out->inst_cap = E + R * ns;
  out->phys = R * c->P;
  out->rank_load = R;
  out->rank_base = R + 1;
  out->U = E * R;
  out->scalars = UEP_N_SCALARS;
  out->M = c->M;
  out->P = c->P;
  return UEP_OK;
}

int uep_get_launch_info(const uep_ctx* ctx, uep_launch_info* out) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !out) return UEP_ERR_INVALID_ARG;
  out->n_chunks = c->n_chunks;
  out->chunk_len = c->chunk_len;
  out->hist_threads = kHistThreads;
  out->remap_threads = kRemapThreads;
  out->plan_threads = kPlanThreads;
  out->pack_ctas = c->pack_ctas;
  out->pack_tile_bytes = kPackTile;
  out->sm_count = c->sm_count;
  out->r_chunks = c->r_chunks;
  out->r_chunk_len = c->r_chunk_len;
  out->plan_cluster = c->plan_cluster;
  return UEP_OK;
}

unsigned long long uep_launch_count(const uep_ctx* ctx) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  return c ? __atomic_load_n(&const_cast<Ctx*>(c)->n_launches, __ATOMIC_RELAXED) : 0ull;
}

int uep_histogram(const uep_ctx* ctx, const int32_t* topk_ids, int32_t* expert_count, void* ws,
                  void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !expert_count || !ws || !aligned16(expert_count) || !aligned16(ws))
    return UEP_ERR_INVALID_ARG;
  if (c->S > 0 && (!topk_ids || !aligned16(topk_ids))) return UEP_ERR_INVALID_ARG;
  return launch_histogram(c, topk_ids, expert_count, ws, static_cast<cudaStream_t>(stream));
}

int uep_plan(const uep_ctx* ctx, const int32_t* expert_count, const uep_plan_out* plan, void* ws,
             void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  (void)ws;
  if (!c || !expert_count || !aligned16(expert_count)) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  return launch_plan(c, expert_count, *plan, static_cast<cudaStream_t>(stream));
}

int uep_remap(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
              const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
              int32_t* out_offset, void* out_gate, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  if (c->S > 0) {
    if (!topk_ids || !out_replica || !out_rank || !out_offset) return UEP_ERR_INVALID_ARG;
    if (!aligned16(topk_ids) || !aligned16(out_replica) || !aligned16(out_rank) ||
        !aligned16(out_offset))
      return UEP_ERR_INVALID_ARG;
  }
  if ((gate == nullptr) != (out_gate == nullptr)) return UEP_ERR_INVALID_ARG;
  if (gate && (c->cfg.gate_dtype == UEP_GATE_NONE || !aligned16(gate) || !aligned16(out_gate)))
    return UEP_ERR_INVALID_ARG;
  return launch_remap(c, topk_ids, gate, *plan, out_replica, out_rank, out_offset, out_gate, ws,
                      static_cast<cudaStream_t>(stream));
}

int uep_plan_batched(const uep_ctx* ctx, int32_t n_inst, const int32_t* expert_count,
                     const uep_plan_out* plan0, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || n_inst < 0 || n_inst > 65535 / 16) return UEP_ERR_INVALID_ARG;
  if (n_inst == 0) return UEP_OK;
  if (!expert_count || !aligned16(expert_count)) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan0);
  if (rc != UEP_OK) return rc;
  return launch_plan(c, expert_count, *plan0, static_cast<cudaStream_t>(stream), false, n_inst);
}

static int check_remap_outputs(const Ctx* c, const void* gate, const uep_plan_out* plan,
                               const int32_t* out_replica, const int32_t* out_rank,
                               const int32_t* out_offset, const void* out_gate, const void* ws) {
  if (!ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  if (c->S > 0) {
    if (!out_replica || !out_rank || !out_offset) return UEP_ERR_INVALID_ARG;
    if (!aligned16(out_replica) || !aligned16(out_rank) || !aligned16(out_offset))
      return UEP_ERR_INVALID_ARG;
  }
  if ((gate == nullptr) != (out_gate == nullptr)) return UEP_ERR_INVALID_ARG;
  if (gate && (c->cfg.gate_dtype == UEP_GATE_NONE || !aligned16(gate) || !aligned16(out_gate)))
    return UEP_ERR_INVALID_ARG;
  return UEP_OK;
}

int uep_remap_rank(const uep_ctx* ctx, const int32_t* topk_ids, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  if (c->S > 0 && (!topk_ids || !aligned16(topk_ids))) return UEP_ERR_INVALID_ARG;
  return launch_rank(c, topk_ids, ws, static_cast<cudaStream_t>(stream));
}

int uep_remap_lookup(const uep_ctx* ctx, const void* gate, const uep_plan_out* plan,
                     int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                     void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  int rc = check_remap_outputs(c, gate, plan, out_replica, out_rank, out_offset, out_gate, ws);
  if (rc != UEP_OK) return rc;
  return launch_lookup(c, gate, *plan, out_replica, out_rank, out_offset, out_gate, ws,
                       static_cast<cudaStream_t>(stream));
}

int uep_pack(const uep_ctx* ctx, const uep_plan_out* plan, int32_t n_tensors,
             const void* const* src, const size_t* bytes_per_expert, void* const* dst,
             void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  PackArgs a;
  rc = fill_pack_args(n_tensors, src, bytes_per_expert, dst, a);
  if (rc != UEP_OK) return rc;
  if (n_tensors == 0 || c->cfg.n_slot == 0) return UEP_OK;
  return launch_pack(c, *plan, a, static_cast<cudaStream_t>(stream));
}

int uep_remap_local(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
                    const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
                    int32_t* out_offset, void* out_gate, int32_t* n_inflight, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  if (c->S > 0 && c->l_cpg == 0) return UEP_ERR_UNSUPPORTED;           // T must be a multiple of R
  int rc = check_remap_outputs(c, gate, plan, out_replica, out_rank, out_offset, out_gate, ws);
  if (rc != UEP_OK) return rc;
  if (c->S > 0 && (!topk_ids || !aligned16(topk_ids))) return UEP_ERR_INVALID_ARG;
  if (n_inflight && !aligned16(n_inflight)) return UEP_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  rc = launch_rank(c, topk_ids, ws, s, /*local=*/true);
  if (rc == UEP_OK) rc = launch_reroute(c, *plan, n_inflight, ws, s);
  if (rc == UEP_OK)
    rc = launch_lookup(c, gate, *plan, out_replica, out_rank, out_offset, out_gate, ws, s, /*pdl=*/true,
                       /*local=*/true, n_inflight);   // prologue overlaps reroute_kernel
  return rc;
}

// ---- token-sharded path ----------------------------------------------------------
// Shard g of G owns source ranks [g*R/G, (g+1)*R/G): chunks [g*cps, (g+1)*cps) of the grouped
// geometry (cps = R/G * l_cpg) and slots [g*S/G, (g+1)*S/G).  The kernels index the GLOBAL slot
// arrays; a shard's local buffers are addressed through a virtual base (local pointer minus the
// shard's first slot) of which only the shard's own range is ever dereferenced.
struct ShardGeom { int chunk0, chunks; long long slot0; };

static int shard_geom(const Ctx* c, int32_t shard, int32_t n_shards, ShardGeom* g) {
  if (n_shards < 1 || shard < 0 || shard >= n_shards || c->cfg.R % n_shards != 0) return UEP_ERR_INVALID_ARG;
  if (c->S > 0 && c->l_cpg == 0) return UEP_ERR_UNSUPPORTED;           // T must be a multiple of R
  const int rps = c->cfg.R / n_shards;
  g->chunks = rps * c->l_cpg;
  g->chunk0 = shard * g->chunks;
  g->slot0 = (long long)shard * rps * c->l_group_len;
  return UEP_OK;
}

static void* virtual_base(const void* local, long long slot0, size_t elem) {
  return local ? reinterpret_cast<void*>(reinterpret_cast<uintptr_t>(local) - (uintptr_t)slot0 * elem) : nullptr;
}

int uep_shard_rows(const uep_ctx* ctx, int32_t shard, int32_t n_shards, size_t* ws_byte_offset,
                   size_t* n_bytes) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !ws_byte_offset || !n_bytes) return UEP_ERR_INVALID_ARG;
  ShardGeom g;
  int rc = shard_geom(c, shard, n_shards, &g);
  if (rc != UEP_OK) return rc;
  // the shard's rows of Lambda[R][E_pad] (one row per source rank: lambda_{r,e})
  const size_t row = sizeof(int32_t) * (size_t)c->E_pad;
  const int rps = c->cfg.R / n_shards;
  *ws_byte_offset = ws_lambda_offset(c) + row * (size_t)(shard * rps);
  *n_bytes = row * (size_t)rps;
  return UEP_OK;
}

int uep_shard_count(const uep_ctx* ctx, int32_t shard, int32_t n_shards,
                    const int32_t* topk_ids_local, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  ShardGeom g;
  int rc = shard_geom(c, shard, n_shards, &g);
  if (rc != UEP_OK) return rc;
  if (c->S == 0) return UEP_OK;
  if (!topk_ids_local || !aligned16(topk_ids_local)) return UEP_ERR_INVALID_ARG;
  // The rows the exchange needs come from one quick counting pass over the shard's ids
  // (shard_hist_kernel -> shard_rows_kernel on `stream`); the stable ranks, which only the lookup of
  // uep_shard_finish needs, are made beside it on the context's side stream (forked here, joined in
  // uep_shard_finish: the same scheme as uep_balance, and the general rank kernel for the same
  // reason).  Before: rank kernel, then the rows from its counts, all in front of the exchange
  // (token-sharded step 35.7 us at G = 1 on the DeepSeek-V3 shape).
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int32_t* vids = static_cast<const int32_t*>(virtual_base(topk_ids_local, g.slot0, 4));
  const int rps = c->cfg.R / n_shards;
  cudaError_t ce = cudaSuccess;
  bool forked = false;
#define UEP_SH_TRY(expr) do { if (rc == UEP_OK && ce == cudaSuccess) ce = (expr); } while (0)
#define UEP_SH_RC(expr) do { if (rc == UEP_OK && ce == cudaSuccess) rc = (expr); } while (0)
  UEP_SH_TRY(cudaEventRecord(c->ev_fork, s));
  UEP_SH_RC(launch_shard_hist(c, vids, ws, s, g.chunk0, g.chunks));       // launched first: its CTAs take the SMs first
  UEP_SH_TRY(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
  forked = (rc == UEP_OK && ce == cudaSuccess);
  UEP_SH_RC(launch_rank(c, vids, ws, c->side, /*local=*/true, g.chunk0, g.chunks, /*with_prefix=*/false,
                        /*bitmaps=*/false, /*write_counts=*/false));
  UEP_SH_TRY(cudaEventRecord(c->ev_rank, c->side));
  UEP_SH_RC(launch_shard_rows(c, ws, s, shard * rps, rps));
#undef UEP_SH_TRY
#undef UEP_SH_RC
  if (rc == UEP_OK && ce == cudaSuccess) return UEP_OK;
  if (ce != cudaSuccess) rc = set_cuda_error(ce);
  if (forked) {                  // join what was forked: an enclosing capture stays valid
    if (cudaEventRecord(c->ev_join, c->side) == cudaSuccess) cudaStreamWaitEvent(s, c->ev_join, 0);
  }
  cudaGetLastError();
  return rc;
}

int uep_shard_finish(const uep_ctx* ctx, int32_t shard, int32_t n_shards, const void* gate_local,
                     int32_t* expert_count, const uep_plan_out* plan, int32_t* out_replica_local,
                     int32_t* out_rank_local, int32_t* out_offset_local, void* out_gate,
                     int32_t* n_inflight, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !expert_count || !aligned16(expert_count)) return UEP_ERR_INVALID_ARG;
  ShardGeom g;
  int rc = shard_geom(c, shard, n_shards, &g);
  if (rc != UEP_OK) return rc;
  rc = check_remap_outputs(c, gate_local, plan, out_replica_local, out_rank_local, out_offset_local,
                           out_gate, ws);
  if (rc != UEP_OK) return rc;
  if (n_inflight && !aligned16(n_inflight)) return UEP_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (c->S == 0) {                                                     // identity plan of an empty batch
    UEP_CUDA_TRY(cudaMemsetAsync(expert_count, 0, sizeof(int32_t) * c->cfg.E, s));
    return launch_plan(c, expert_count, *plan, s);
  }
  const int rps = c->cfg.R / n_shards;
  // lambda_e = the column sums of the gathered Lambda: the planner adds them up itself and publishes
  // expert_count; planner and lookup are programmatically dependent on their predecessors.  The lookup
  // derives the GLOBAL rank base of each of its chunks from Lambda and its own chunk counts in its
  // prologue, beside the planner: no kernel between the exchange and the planner
  rc = launch_plan(c, nullptr, *plan, s, /*pdl=*/true, 1, ws_lambda(c, ws), expert_count, c->cfg.R, c->E_pad,
                   n_inflight ? n_inflight + shard * rps : nullptr, n_inflight ? rps : 0);
  const size_t gb = c->cfg.gate_dtype == UEP_GATE_BF16 ? 2 : 4;
  // join the rank kernel that uep_shard_count left on the side stream (also when the planner's launch
  // failed: a capture must not end with an un-joined fork)
  if (cudaStreamWaitEvent(s, c->ev_rank, 0) != cudaSuccess && rc == UEP_OK) rc = set_cuda_error(cudaGetLastError());
  if (rc == UEP_OK)
    rc = launch_lookup(c, virtual_base(gate_local, g.slot0, gb), *plan,
                       static_cast<int32_t*>(virtual_base(out_replica_local, g.slot0, 4)),
                       static_cast<int32_t*>(virtual_base(out_rank_local, g.slot0, 4)),
                       static_cast<int32_t*>(virtual_base(out_offset_local, g.slot0, 4)), out_gate, ws, s, /*pdl=*/true,
                       /*local=*/true, n_inflight, nullptr, g.chunk0, g.chunks, /*src_aware=*/false,
                       /*from_lambda=*/true);
  return rc;
}

int uep_grad_reduce(const uep_ctx* ctx, const uep_plan_out* plan, int32_t n_tensors,
                    void* const* main_grad, const size_t* bytes_per_expert, void* const* slot_grad,
                    void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  if (n_tensors < 0 || n_tensors > UEP_MAX_TENSORS) return UEP_ERR_INVALID_ARG;
  if (n_tensors && (!main_grad || !bytes_per_expert || !slot_grad)) return UEP_ERR_INVALID_ARG;
  for (int j = 0; j < n_tensors; ++j) {
    if (!main_grad[j] || !slot_grad[j] || !aligned16(main_grad[j]) || !aligned16(slot_grad[j]))
      return UEP_ERR_INVALID_ARG;
    if (bytes_per_expert[j] == 0 || (bytes_per_expert[j] & 15)) return UEP_ERR_INVALID_ARG;
  }
  if (n_tensors == 0 || c->cfg.n_slot == 0) return UEP_OK;
  return launch_grad_reduce(c, *plan, n_tensors, main_grad, slot_grad, bytes_per_expert,
                            static_cast<cudaStream_t>(stream));
}

int uep_relay_plan(const uep_ctx* ctx, const uep_plan_out* plan, int32_t* relay_parent,
                   int32_t* send_volume, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !relay_parent || !send_volume || !aligned16(relay_parent) || !aligned16(send_volume))
    return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  return launch_relay(c, *plan, relay_parent, send_volume, static_cast<cudaStream_t>(stream));
}

int uep_remap_inverse(const uep_ctx* ctx, const int32_t* out_rank, const int32_t* out_offset,
                      const uep_plan_out* plan, int32_t* out_src, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  int rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  if (c->S > 0 && (!out_rank || !out_offset || !out_src || !aligned16(out_rank) ||
                   !aligned16(out_offset) || !aligned16(out_src)))
    return UEP_ERR_INVALID_ARG;
  return launch_inverse(c, out_rank, out_offset, *plan, out_src, static_cast<cudaStream_t>(stream));
}

}  // extern "C"

// uep_balance proper.  join_pack = false leaves the side stream (pack) un-joined: the caller
// enqueues more work on `stream` first and then waits on ctx->ev_join itself (uep_balance_host
// overlaps its device->host copies with the pack that way).
static int balance_impl(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
                        int32_t* expert_count, const uep_plan_out* plan, int32_t* out_replica,
                        int32_t* out_rank, int32_t* out_offset, void* out_gate, int32_t n_tensors,
                        const void* const* src, const size_t* bytes_per_expert, void* const* dst,
                        void* ws, void* stream, bool join_pack) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c) return UEP_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  PackArgs a;
  int rc = fill_pack_args(n_tensors, src, bytes_per_expert, dst, a);
  if (rc != UEP_OK) return rc;
  // argument checks of the remap stage up front: the rank kernel is launched first
  if (!ws || !aligned16(ws)) return UEP_ERR_INVALID_ARG;
  rc = check_plan_ptrs(c, plan);
  if (rc != UEP_OK) return rc;
  if (c->S > 0) {
    if (!topk_ids || !out_replica || !out_rank || !out_offset) return UEP_ERR_INVALID_ARG;
    if (!aligned16(topk_ids) || !aligned16(out_replica) || !aligned16(out_rank) ||
        !aligned16(out_offset))
      return UEP_ERR_INVALID_ARG;
  }
  if ((gate == nullptr) != (out_gate == nullptr)) return UEP_ERR_INVALID_ARG;
  if (gate && (c->cfg.gate_dtype == UEP_GATE_NONE || !aligned16(gate) || !aligned16(out_gate)))
    return UEP_ERR_INVALID_ARG;
  if (!expert_count || !aligned16(expert_count)) return UEP_ERR_INVALID_ARG;
  // fork: the plan-independent half of the remap (stable ranks inside each chunk) runs on the side
  // stream beside histogram + plan.  The histogram is LAUNCHED first (the fork event precedes it,
  // so the rank kernel does not depend on it): its CTAs take the SMs first, the rank CTAs fill in
  // as they retire and run beside the plan.  Measured on B200 (DSV3 shape, whole chain):
  // rank launched first 58.9 us, histogram first 54.5 us, rank made dependent on the histogram
  // 62.5 us (its CTAs then race the plan's cluster for SMs).  Re-measured with the planner
  // launched at high priority (chain 32.2 us): rank made dependent on the histogram 32.7 us.
  // From the first event record on, every failure goes through `fail`: the side stream is joined
  // back into `stream` (a capture stays valid and ends with no un-joined fork) and the histogram's
  // accumulator, which only a completed chain leaves zero, is cleared.
  cudaError_t ce = cudaSuccess;
  bool forked = false;
  rc = UEP_OK;
#define UEP_BAL_TRY(expr) do { if (rc == UEP_OK && ce == cudaSuccess) ce = (expr); } while (0)
#define UEP_BAL_RC(expr) do { if (rc == UEP_OK && ce == cudaSuccess) rc = (expr); } while (0)
  UEP_BAL_TRY(cudaEventRecord(c->ev_fork, s));
  UEP_BAL_RC(launch_histogram(c, topk_ids, expert_count, ws, s, /*red=*/true));
  UEP_BAL_TRY(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
  forked = (rc == UEP_OK && ce == cudaSuccess);
  UEP_BAL_RC(launch_rank(c, topk_ids, ws, c->side, /*local=*/false, 0, -1, /*with_prefix=*/true, /*bitmaps=*/false));
  UEP_BAL_TRY(cudaEventRecord(c->ev_rank, c->side));
  // planner and lookup are launched programmatically dependent on their predecessor: their
  // prologues (static layout; packed ranks, gates) overlap it
  UEP_BAL_RC(launch_plan(c, expert_count, *plan, s, /*pdl=*/true, 1, ws_acc(ws), expert_count));
  const bool do_pack = n_tensors > 0 && c->cfg.n_slot > 0;
  if (do_pack) {   // pack depends only on the plan and overlaps the lookup (Eq. 1)
    UEP_BAL_TRY(cudaEventRecord(c->ev_fork, s));
    UEP_BAL_TRY(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
    UEP_BAL_RC(launch_pack(c, *plan, a, c->side));
  }
  UEP_BAL_TRY(cudaEventRecord(c->ev_join, c->side));
  UEP_BAL_TRY(cudaStreamWaitEvent(s, c->ev_rank, 0));          // join the rank kernel
  UEP_BAL_RC(launch_lookup(c, gate, *plan, out_replica, out_rank, out_offset, out_gate, ws, s, /*pdl=*/true,
                           false, nullptr, ws_acc(ws)));
  if (join_pack) UEP_BAL_TRY(cudaStreamWaitEvent(s, c->ev_join, 0));   // join the side stream (pack)
#undef UEP_BAL_TRY
#undef UEP_BAL_RC
  if (rc == UEP_OK && ce == cudaSuccess) return UEP_OK;
  // ---- failure: join whatever was forked, leave the workspace reusable -----------------------------
  if (ce != cudaSuccess) rc = set_cuda_error(ce);
  if (forked) {
    if (cudaEventRecord(c->ev_join, c->side) == cudaSuccess) cudaStreamWaitEvent(s, c->ev_join, 0);
  }
  cudaMemsetAsync(ws_acc(ws), 0, sizeof(int32_t) * UEP_MAX_E, s);    // a half-run chain may have left counts there
  cudaGetLastError();
  return rc;
}

extern "C" {

int uep_balance(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
                int32_t* expert_count, const uep_plan_out* plan, int32_t* out_replica,
                int32_t* out_rank, int32_t* out_offset, void* out_gate, int32_t n_tensors,
                const void* const* src, const size_t* bytes_per_expert, void* const* dst,
                void* ws, void* stream) {
  return balance_impl(ctx, topk_ids, gate, expert_count, plan, out_replica, out_rank, out_offset,
                      out_gate, n_tensors, src, bytes_per_expert, dst, ws, stream, true);
}

int uep_balance_host(const uep_ctx* ctx, const int32_t* topk_ids_host, const void* gate_host,
                     int32_t* dev_topk_ids, void* dev_gate, int32_t* expert_count,
                     const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
                     int32_t* out_offset, void* out_gate, int32_t* out_replica_host,
                     int32_t* out_rank_host, int32_t* out_offset_host, void* out_gate_host,
                     int32_t* scalars_host, int32_t n_tensors, const void* const* src,
                     const size_t* bytes_per_expert, void* const* dst, void* ws, void* stream) {
  const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
  if (!c || !topk_ids_host || !dev_topk_ids || !plan) return UEP_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t S = (size_t)c->S;
  const size_t gb = c->cfg.gate_dtype == UEP_GATE_F32 ? 4 : (c->cfg.gate_dtype == UEP_GATE_BF16 ? 2 : 0);
  UEP_CUDA_TRY(cudaMemcpyAsync(dev_topk_ids, topk_ids_host, S * 4, cudaMemcpyHostToDevice, s));
  const bool has_gate = gate_host && dev_gate && gb;
  if (has_gate) UEP_CUDA_TRY(cudaMemcpyAsync(dev_gate, gate_host, S * gb, cudaMemcpyHostToDevice, s));
  // the pack (side stream) is joined only after the device->host copies are enqueued: the copies
  // of the remap outputs run over PCIe while the pack streams HBM
  int rc = balance_impl(ctx, dev_topk_ids, has_gate ? dev_gate : nullptr, expert_count, plan,
                        out_replica, out_rank, out_offset, has_gate ? out_gate : nullptr, n_tensors,
                        src, bytes_per_expert, dst, ws, stream, /*join_pack=*/false);
  if (rc != UEP_OK) { cudaStreamWaitEvent(s, c->ev_join, 0); return rc; }
  if (out_replica_host) UEP_CUDA_TRY(cudaMemcpyAsync(out_replica_host, out_replica, S * 4, cudaMemcpyDeviceToHost, s));
  if (out_rank_host) UEP_CUDA_TRY(cudaMemcpyAsync(out_rank_host, out_rank, S * 4, cudaMemcpyDeviceToHost, s));
  if (out_offset_host) UEP_CUDA_TRY(cudaMemcpyAsync(out_offset_host, out_offset, S * 4, cudaMemcpyDeviceToHost, s));
  if (has_gate && out_gate_host) UEP_CUDA_TRY(cudaMemcpyAsync(out_gate_host, out_gate, S * gb, cudaMemcpyDeviceToHost, s));
  if (scalars_host) UEP_CUDA_TRY(cudaMemcpyAsync(scalars_host, plan->scalars, sizeof(int32_t) * UEP_N_SCALARS, cudaMemcpyDeviceToHost, s));
  UEP_CUDA_TRY(cudaStreamWaitEvent(s, c->ev_join, 0));          // join the side stream (pack)
  UEP_CUDA_TRY(cudaStreamSynchronize(s));
  return UEP_OK;
}

const char* uep_strerror(int code) {
  switch (code) {
    case UEP_OK: return "ok";
    case UEP_ERR_INVALID_ARG: return "invalid argument (NULL or misaligned pointer, bad size)";
    case UEP_ERR_UNSUPPORTED: return "unsupported shape or device (limits in uep.h; sm_100 required)";
    case UEP_ERR_CUDA: return "CUDA error (see uep_last_cuda_error)";
    case UEP_ERR_NO_DEVICE: return "no CUDA device";
    default: return "unknown error";
  }
}

const char* uep_last_cuda_error(void) { return g_cuda_err; }

}  // extern "C"
