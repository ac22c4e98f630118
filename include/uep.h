/* uep.h — C ABI of libuep: the post-gating, exact-load balance-planning step of UltraEP
 * (arxiv 2606.04101), emulated for R virtual expert-parallel ranks on ONE B200 (sm_100a).
 *
 *   uep_histogram : lambda_e, the per-expert token load              (Alg. 1 line 2)
 *   uep_plan      : SolveReplication, quota-driven planner           (Alg. 1 lines 1-25, PAPER.md:247-297;
 *                                                                     §5.1; §5.3)
 *   uep_remap     : token assignment by cumulative-quota lookup      (§5.2 "Token Assignment")
 *   uep_pack      : weight distribution main -> redundant slot,      (§4.2, §6.1)
 *                   single-GPU part: pack into per-destination buffers
 *   uep_balance   : the four chained on one stream, capturable in a CUDA graph
 *                   ("fully on-device ... preserves the graph capture")
 *
 * Conventions (all entry points)
 *   - plain C; every pointer argument says HOST or DEVICE below; `stream` is a cudaStream_t
 *     passed as void* so that this header needs no CUDA include.
 *   - return 0 (UEP_OK) or a negative UEP_ERR_*; uep_strerror() gives the text.
 *   - after uep_create: asynchronous on `stream`, no host synchronisation, no allocation,
 *     no host memory touched => every compute call can be stream-captured.
 *   - ownership: the library never frees or retains caller pointers beyond the call.
 *     Outputs and workspace are caller-allocated DEVICE memory.  A context may be shared by
 *     concurrent calls of uep_histogram / uep_plan / uep_remap* / uep_pack on different streams;
 *     a workspace may not (one per in-flight call).  uep_balance uses the context's internal
 *     side stream and events: calls of uep_balance on one context must be issued from one host
 *     thread at a time (they may target different streams; create one context per concurrent
 *     host thread).  uep_pack / uep_grad_reduce take their work counter from a pool of 64 the
 *     context owns (round robin, self-resetting): at most 64 such kernels of one context may be
 *     executing at the same time, and one captured graph must not be replayed concurrently with
 *     itself.
 *   - data faults that would need a sync to report (an id outside [0,E)) are counted on the
 *     device (scalars[UEP_SC_N_INVALID]) and the slot is skipped (S14).
 *   - all DEVICE pointers must be 16-byte aligned.
 *
 * Notation (Table 1): E logical experts, R ranks, N_slot redundant slots per
 * rank, h(e) home rank, lambda_e load, l_r initial rank load, U quotas, X slot assignment.
 * S = T*k routed slots; M = max_r |E_r| main slots per rank; P = M + N_slot physical slots.
 */
#ifndef UEP_H_
#define UEP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define UEP_MAX_E 512        /* shared-memory histogram / planner tables are sized for this */
#define UEP_MAX_R 256
#define UEP_MAX_NSLOT 4
#define UEP_MAX_TENSORS 8

enum { UEP_FLOOR_STRICT = 0,     /* Alg. 1 line 20 verbatim: feasible iff sum_r exc_r == 0      */
       UEP_FLOOR_TOLERANT = 1 }; /* DESIGN.md S8 (default): feasible iff every exc_r < u_min    */
enum { UEP_GATE_F32 = 0, UEP_GATE_BF16 = 1, UEP_GATE_NONE = 2 };

enum { UEP_OK = 0,
       UEP_ERR_INVALID_ARG = -1,   /* NULL / misaligned pointer, bad size                        */
       UEP_ERR_UNSUPPORTED = -2,   /* shape outside the limits above                             */
       UEP_ERR_CUDA = -3,          /* a CUDA runtime call or launch failed                       */
       UEP_ERR_NO_DEVICE = -4 };

/* plan->scalars[] indices (int32 each, UEP_N_SCALARS entries) */
enum { UEP_SC_TAU = 0,           /* final threshold tau (Alg. 1: tau_hi on exit)                 */
       UEP_SC_N_REPLICAS = 1,    /* number of redundant slots used, sum_e (|H(e)|-1)             */
       UEP_SC_MAX_LOAD = 2,      /* max_r sum_e u_{e,r}                      (Eq. 3) */
       UEP_SC_MAX_FANOUT = 3,    /* max_e |H(e)|                              (Table 3)           */
       UEP_SC_N_PROBES = 4,      /* probes on the sequential bisection path                      */
       UEP_SC_N_INVALID = 5,     /* T*k - sum_e lambda_e                                         */
       UEP_SC_TAU_LO0 = 6,       /* tau_lo on entry                                              */
       UEP_SC_TAU_HI0 = 7,       /* tau_hi on entry = max_r l_r                                  */
       UEP_SC_N_GROUPS = 8,      /* number of experts with at least one replica                  */
       UEP_N_SCALARS = 16 };

/* Opaque.  Shapes, launch geometry and the static layout are immutable after uep_create.  The
 * context also owns a little MUTABLE launch state: the internal side stream and three events that
 * uep_balance forks and joins on, a round-robin index into the work-counter pool of uep_pack /
 * uep_grad_reduce, and a launch counter (uep_launch_count) — see the threading rules above. */
typedef struct uep_ctx uep_ctx;

typedef struct uep_config {
  int32_t T, k;                  /* tokens and top-k; S = T*k < 2^24 slots (S20: the
                                    planner packs a rank's slack into 24 bits of its arg-max key;
                                    the BASELINE configs reach 2^22)                              */
  int32_t E, R, n_slot;          /* 1<=E<=512, 1<=R<=256, 0<=n_slot<=4                            */
  int32_t u_min;                 /* quota floor u_min >= 1 (paper: 1024)           */
  int32_t beta_num, beta_den;    /* balancing target beta as a rational (paper: 101/100)         */
  int32_t floor_mode;            /* UEP_FLOOR_*                                                   */
  int32_t gate_dtype;            /* UEP_GATE_*                                                    */
  const int32_t* home_rank;      /* HOST [E] or NULL => h(e) = floor(e*R/E)        (S2) */
} uep_config;

/* element counts (int32 elements) of every plan array, plus the derived M and P */
typedef struct uep_plan_sizes {
  int32_t slot_expert;           /* R*n_slot (>=1 allocated)                                      */
  int32_t inst_off;              /* E+1                                                           */
  int32_t inst_cap;              /* E + R*n_slot : inst_rank / inst_phys / inst_cum / inst_base   */
  int32_t phys;                  /* R*P : phys_count / phys_base                                  */
  int32_t rank_load;             /* R                                                             */
  int32_t rank_base;             /* R+1                                                           */
  int32_t U;                     /* E*R (optional dense quota table)                              */
  int32_t scalars;               /* UEP_N_SCALARS                                                 */
  int32_t M, P;
} uep_plan_sizes;

/* The plan: a struct (in HOST memory) of DEVICE pointers, all int32.
 *   slot_expert[R][n_slot]  X: expert replicated in redundant slot s of rank t, -1 = empty;
 *                           used slots of a rank are a prefix, in acceptance order (S10)
 *   inst_off[E+1]           CSR over logical experts into the instance arrays
 *   inst_rank/phys/cum[]    instances of e in order [main, replicas in acceptance order] (S11):
 *                           host rank, local physical slot on that rank (main e -> its index
 *                           among E_{h(e)} ascending; redundant slot s -> M+s), and the
 *                           INCLUSIVE cumulative quota (last = lambda_e)
 *   inst_base[]             offset of the instance's first token inside its host rank's receive
 *                           buffer = phys_base[inst_rank][inst_phys] (S13), same indexing
 *   phys_count/base[R][P]   tokens received per local physical slot and their exclusive prefix
 *   rank_load[R]            sum_e u_{e,t};  rank_base[R+1] its exclusive prefix (last = #valid)
 *   scalars[UEP_N_SCALARS]  see UEP_SC_*
 *   U[E][R]                 dense quota table, may be NULL (tests / inspection only)        */
typedef struct uep_plan_out {
  int32_t* slot_expert;
  int32_t* inst_off;
  int32_t* inst_rank;
  int32_t* inst_phys;
  int32_t* inst_cum;
  int32_t* inst_base;
  int32_t* phys_count;
  int32_t* phys_base;
  int32_t* rank_load;
  int32_t* rank_base;
  int32_t* scalars;
  int32_t* U;
} uep_plan_out;

/* Create a context for fixed shapes (validates limits, uploads the static layout h(e), E_r,
 * main slot indices).  cfg: HOST.  Uses the current CUDA device.  Allocates a few KB of
 * device memory, freed by uep_destroy. */
int uep_create(const uep_config* cfg, uep_ctx** out);
void uep_destroy(uep_ctx* ctx);

/* Bytes of DEVICE workspace one in-flight call needs (scratch of the histogram's chunk table,
 * and of the remap: per-chunk expert counts, their exclusive prefix over chunks and one packed
 * int32 {expert, rank inside chunk} per slot, ~4 bytes per slot in total).
 * uep_workspace_init must be called once (async on `stream`) before first use: it zeroes the
 * histogram's accumulator and the first row of the remap's prefix table, which every call then
 * leaves zero again.  (A departure from the header SURVEY.md §8(b) proposed, which had no such
 * call: the alternative is a memset node in every uep_balance.) */
size_t uep_workspace_bytes(const uep_ctx* ctx);
int uep_workspace_init(const uep_ctx* ctx, void* ws, void* stream);
int uep_plan_bytes(const uep_ctx* ctx, uep_plan_sizes* out);      /* out: HOST */

/* lambda_e = #{slots s : topk_ids[s] == e} (Alg. 1 line 2).
 *   topk_ids      DEVICE int32 [T,k] row-major (slot s = i*k + kk)
 *   expert_count  DEVICE int32 [E], overwritten
 *   ws            DEVICE workspace (initialised); scratch: an accumulator that the call leaves
 *                 zero again, and the per-CTA count rows.  Two kernels, the second one launched
 *                 programmatically dependent on the first; asynchronous, capturable.          */
int uep_histogram(const uep_ctx* ctx, const int32_t* topk_ids, int32_t* expert_count, void* ws,
                  void* stream);

/* SolveReplication (Alg. 1 lines 1-25) under the readings of DESIGN.md §3; emits X, U (as CSR
 * cumulative quotas) and the receive layout.  expert_count: DEVICE int32 [E].  plan: HOST struct
 * of DEVICE pointers (U may be NULL).  ws is not modified. */
int uep_plan(const uep_ctx* ctx, const int32_t* expert_count, const uep_plan_out* plan, void* ws,
             void* stream);

/* Batched SolveReplication: n_inst independent instances (layers x microbatches whose loads are
 * known together, e.g. replay or simulation as in Fig. 15) in ONE launch, one
 * thread-block cluster per instance, all clusters concurrent on different SMs.
 *   expert_count  DEVICE int32 [n_inst][E]
 *   plan0         HOST struct of DEVICE pointers to the arrays of instance 0; every array must be
 *                 allocated n_inst times its uep_plan_sizes element count, instance b starting
 *                 b * count elements after instance 0 (U may be NULL).
 * Each instance's result is bit-identical to uep_plan on its counts. */
int uep_plan_batched(const uep_ctx* ctx, int32_t n_inst, const int32_t* expert_count,
                     const uep_plan_out* plan0, void* stream);

/* Token assignment (§5.2): slot s of expert e with global stable rank j goes to the first
 * instance whose cumulative quota exceeds j.
 *   gate          DEVICE [T,k] of cfg.gate_dtype, or NULL
 *   out_replica/out_rank/out_offset  DEVICE int32 [T,k]; (-1,-1,-1) for an invalid id
 *   out_gate      DEVICE [T*k] gate dtype, written at rank_base[rank]+offset (raw bit copy);
 *                 positions past the number of valid slots are not written
 *   ws            scratch of this call (chunk ranks and their prefix over chunks); the plan must
 *                 have been computed from the histogram of the SAME topk_ids                 */
int uep_remap(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
              const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
              int32_t* out_offset, void* out_gate, void* ws, void* stream);

/* The two halves of uep_remap, for callers that overlap them with other work (uep_balance does):
 *   uep_remap_rank    plan-INDEPENDENT: stable rank of every slot among the slots of its expert
 *                     inside its chunk, written to the workspace.  Needs only topk_ids; may run
 *                     concurrently with uep_histogram / uep_plan on another stream.
 *   uep_remap_lookup  plan-DEPENDENT: needs ws after uep_remap_rank on the same topk_ids, and
 *                     the plan of those ids.  Same outputs and argument rules as uep_remap.
 * uep_remap(...) == uep_remap_rank(...) then uep_remap_lookup(...) on one stream.
 * uep_remap_rank accepts any ids.  When every token names an expert at most once (what top-k
 * routing produces) and 2 <= k <= 64 it ranks with per-expert token bitmaps, which is faster; a
 * token that repeats an expert sends its chunk through the general method.  Same result either way. */
int uep_remap_rank(const uep_ctx* ctx, const int32_t* topk_ids, void* ws, void* stream);
int uep_remap_lookup(const uep_ctx* ctx, const void* gate, const uep_plan_out* plan,
                     int32_t* out_replica, int32_t* out_rank, int32_t* out_offset, void* out_gate,
                     void* ws, void* stream);

/* Source-aware reroute and token assignment (SolveReroute, Alg. 1 lines 26-36, PAPER.md:298-320;
 * §5.2).  Token i belongs to source rank floor(i*R/T) (S1).  For every
 * expert the solved quotas U are decomposed into q[r,e,t]: every host rank first consumes its own
 * quota (line 29), the residual demand is spread over the residual quotas by the number-line
 * overlap of DESIGN.md S18 (both marginals exact).  The j-th local slot of (r, e) goes to the first
 * instance whose cumulative q[r,e,.] covers j; inside an instance tokens arrive ordered by source
 * rank, then local order (S25), so (rank, offset) is again a bijection onto the receive buffers.
 * Same arguments as uep_remap, plus
 *   n_inflight  DEVICE int32 [R] or NULL: slots of source rank r sent to another rank.
 * Needs T % R == 0 (else UEP_ERR_UNSUPPORTED).  Runs four kernels on `stream`; ws as for uep_remap. */
int uep_remap_local(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
                    const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
                    int32_t* out_offset, void* out_gate, int32_t* n_inflight, void* ws, void* stream);

/* Token-sharded path for G real GPUs (§4.2 "each rank computes gating for its local tokens ...
 * exchanges the count matrix ... every rank solves the same plan").
 * GPU g of G (G divides R, T % R == 0) owns the tokens of source ranks [g*R/G, (g+1)*R/G), i.e.
 * the contiguous slot range [g*S/G, (g+1)*S/G).  One layer is
 *   uep_shard_count   on every GPU: one counting pass over its LOCAL slots leaves this shard's rows
 *                     of the count matrix Lambda[R][E] (lambda_{r,e}: one row of E_pad int32 per
 *                     source rank the shard owns) in ws, on `stream`; the stable ranks of the slots,
 *                     which only uep_shard_finish needs, are computed beside it on the context's
 *                     internal side stream (forked from `stream` here);
 *   an all-gather     of those rows, by the caller (NCCL / torch.distributed; the only exchange:
 *                     4 * E_pad * R bytes in total, 64 KB at R = 64, E = 256).  uep_shard_rows gives
 *                     the byte range of shard g's rows inside ws: the ranges of shards 0..G-1 are
 *                     equal-sized, contiguous and in shard order, so an in-place all-gather on
 *                     ws[offset(0) .. offset(0) + G*bytes) does it.  With G = 1 there is nothing to
 *                     exchange and count -> finish is one capturable sequence;
 *   uep_shard_finish  on every GPU, redundantly and deterministically: exclusive prefix of Lambda over
 *                     source ranks (+ the shard's own per-chunk counts) = the GLOBAL stable rank base
 *                     of every local chunk, lambda_e = the column sums -> expert_count, the SAME plan
 *                     everywhere, then the lookup of the local slots.
 * The concatenation of the shards' outputs equals uep_remap on the whole input (global stable
 * order, S12), bit for bit; G = 1 is the whole problem.
 *   topk_ids_local / gate_local / out_*_local   DEVICE, the shard's S/G slots, 16-B aligned
 *   out_gate     DEVICE [T*k], GLOBAL dispatch order: only the entries of this shard's slots are
 *                written (in the deployment the dispatch carries the gate with the token)
 *   n_inflight   DEVICE int32 [R] or NULL: entries of this shard's source ranks are set to the
 *                number of their slots that leave the rank
 *   ws           sized by uep_workspace_bytes (of the whole problem), initialised once
 * uep_shard_finish joins the side stream's work in front of its lookup, so the pair uses the context's
 * side stream and events like uep_balance: issue uep_shard_count / uep_shard_finish of one context from
 * one host thread at a time, call them on the SAME `stream`, and under stream capture put both into
 * the same capture (a capture that ends after uep_shard_count alone ends with an un-joined fork).
 * Errors: UEP_ERR_UNSUPPORTED if T % R != 0; UEP_ERR_INVALID_ARG if G does not divide R, g is
 * out of range, or a pointer is NULL / misaligned. */
int uep_shard_count(const uep_ctx* ctx, int32_t shard, int32_t n_shards,
                    const int32_t* topk_ids_local, void* ws, void* stream);
int uep_shard_rows(const uep_ctx* ctx, int32_t shard, int32_t n_shards, size_t* ws_byte_offset,
                   size_t* n_bytes);
int uep_shard_finish(const uep_ctx* ctx, int32_t shard, int32_t n_shards, const void* gate_local,
                     int32_t* expert_count, const uep_plan_out* plan, int32_t* out_replica_local,
                     int32_t* out_rank_local, int32_t* out_offset_local, void* out_gate,
                     int32_t* n_inflight, void* ws, void* stream);

/* Pack the state of every replicated expert into its destination slot:
 *   dst[j][(t*n_slot+s)*B_j .. +B_j) = src[j][e*B_j .. +B_j)  for x_{t,s} = e != empty.
 * Empty slots are not touched.  src/dst/bytes_per_expert: HOST arrays [n_tensors] of DEVICE
 * pointers / sizes; B_j % 16 == 0; n_tensors <= UEP_MAX_TENSORS. */
int uep_pack(const uep_ctx* ctx, const uep_plan_out* plan, int32_t n_tensors,
             const void* const* src, const size_t* bytes_per_expert, void* const* dst,
             void* stream);

/* Backward gradient reduction (§4.2, §6.1), single-GPU part: for every
 * replicated expert e, main_grad[j][e] += sum of slot_grad[j][t][s] over its replicas (t,s) in
 * instance order (fp32, bit-reproducible), and those slot buffers are cleared in place; empty
 * slots are not touched.  main_grad/slot_grad/bytes_per_expert: HOST arrays [n_tensors] of DEVICE
 * float pointers ([E, B_j/4] and [R, n_slot, B_j/4]) and sizes B_j in bytes, B_j % 16 == 0. */
int uep_grad_reduce(const uep_ctx* ctx, const uep_plan_out* plan, int32_t n_tensors,
                    void* const* main_grad, const size_t* bytes_per_expert, void* const* slot_grad,
                    void* stream);

/* Load-aware relay scheduling, topology only (§6.2): for every expert with more
 * than 4 replicas, sqrt(f) (to nearest) first-stage relays among its replica ranks with the
 * smallest sending volume, the other replicas attached to the relay whose volume would remain
 * smallest; experts are processed in ascending id, volumes updated in between (S24).
 *   relay_parent  DEVICE int32 [E + R*n_slot], aligned with the plan's CSR: -1 for main instances
 *                 and unused entries, else the rank that sends this replica its copy
 *   send_volume   DEVICE int32 [R]: copies each rank sends under the resulting trees          */
int uep_relay_plan(const uep_ctx* ctx, const uep_plan_out* plan, int32_t* relay_parent,
                   int32_t* send_volume, void* stream);

/* Reverse reroute ("a scatter-to-gather inversion of the forward assignment"):
 * out_src[rank_base[rank[s]] + offset[s]] = s for every valid slot s (the gather list of the
 * combine step / backward dispatch); positions past the number of valid slots are -1.
 *   out_rank/out_offset  DEVICE int32 [T,k] as written by uep_remap;  out_src  DEVICE int32 [T*k] */
int uep_remap_inverse(const uep_ctx* ctx, const int32_t* out_rank, const int32_t* out_offset,
                      const uep_plan_out* plan, int32_t* out_src, void* stream);

/* histogram -> plan -> remap and pack, chained on `stream`.  Internally forked/joined with
 * events on a side stream: uep_remap_rank runs beside histogram + plan (it does not depend on
 * them), and pack runs beside uep_remap_lookup, overlapping the reroute with the weight
 * distribution as in Eq. 1, max(T_reroute, T_w_distr).  Capturable.
 * n_tensors may be 0.  If a launch fails part-way (UEP_ERR_CUDA / UEP_ERR_UNSUPPORTED from a
 * stage), the side stream is joined back into `stream` before returning, so an enclosing stream
 * capture stays valid, and the workspace's accumulator is cleared: the workspace can be reused. */
int uep_balance(const uep_ctx* ctx, const int32_t* topk_ids, const void* gate,
                int32_t* expert_count, const uep_plan_out* plan, int32_t* out_replica,
                int32_t* out_rank, int32_t* out_offset, void* out_gate, int32_t n_tensors,
                const void* const* src, const size_t* bytes_per_expert, void* const* dst,
                void* ws, void* stream);

/* Convenience for callers with HOST buffers (the bench's end-to-end leg): copies ids/gate to
 * the device buffers in `dev_*`, runs uep_balance, copies the remap outputs and the scalars
 * back, and synchronises `stream`.  Host buffers should be pinned.  Expert state stays resident. */
int uep_balance_host(const uep_ctx* ctx, const int32_t* topk_ids_host, const void* gate_host,
                     int32_t* dev_topk_ids, void* dev_gate, int32_t* expert_count,
                     const uep_plan_out* plan, int32_t* out_replica, int32_t* out_rank,
                     int32_t* out_offset, void* out_gate, int32_t* out_replica_host,
                     int32_t* out_rank_host, int32_t* out_offset_host, void* out_gate_host,
                     int32_t* scalars_host, int32_t n_tensors, const void* const* src,
                     const size_t* bytes_per_expert, void* const* dst, void* ws, void* stream);

/* Histogram for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same lambda_e as uep_histogram (Alg. 1 line 2,
 * PAPER.md:250; ids outside [0,E) skipped, S14) with NO context and NO workspace.  The
 * per-CTA count rows that uep_histogram keeps in the caller's workspace live in a fixed array in
 * the library's device image (192 rows x UEP_MAX_E int32 = 384 KB on every GPU that loads the
 * library, until the process exits).  The call allocates nothing: no cudaMalloc / cudaFree and no
 * allocating library routine, on the first call or later.
 *   topk_ids      DEVICE int32 [n_slots], 16-byte aligned (may be NULL when n_slots == 0)
 *   n_slots       0 .. UEP_STATIC_MAX_SLOTS; beyond it UEP_ERR_UNSUPPORTED, nothing launched
 *   E             1 .. UEP_MAX_E; outside it UEP_ERR_UNSUPPORTED, nothing launched
 *   expert_count  DEVICE int32 [E], out, 16-byte aligned
 * Two kernels on `stream` of the CURRENT device, asynchronous.  uep_static_last_error() gives the
 * text of the last rejection on this thread (which limit, which value).  The first call on a device
 * resolves the array's address there (cudaGetSymbolAddress, once per device); make that call — or
 * uep_histogram_static_setup(), with the device current — outside stream capture.
 * ALL calls on a device share the one array, and it keeps the last call's rows (every row a call
 * reads it has written itself, nothing needs clearing): calls that OVERLAP on the GPU — different
 * streams without an ordering between them, or a graph replayed concurrently with itself — race.
 * Calls ordered on one stream, or by events, are safe. */
#define UEP_STATIC_MAX_SLOTS (1 << 24)
int uep_histogram_static_setup(void);
int uep_histogram_static(const int32_t* topk_ids, long long n_slots, int32_t E, int32_t* expert_count,
                         void* stream);
const char* uep_static_last_error(void);

/* Number of kernels launched through this context so far (host-side count, all entry points).
 * The bench reports the difference over its timed region as gpu_launches. */
unsigned long long uep_launch_count(const uep_ctx* ctx);

const char* uep_strerror(int code);
const char* uep_last_cuda_error(void);   /* text of the last CUDA error seen on this thread */

/* Launch geometry chosen at create time, for the bench's roofline arithmetic. */
typedef struct uep_launch_info {
  int32_t n_chunks, chunk_len;   /* histogram: CTAs and slots per CTA                           */
  int32_t hist_threads, remap_threads, plan_threads, pack_ctas, pack_tile_bytes, sm_count;
  int32_t r_chunks, r_chunk_len; /* remap (rank + lookup kernels): CTAs and slots per CTA       */
  int32_t plan_cluster;          /* CTAs (thread-block cluster size) sharing one plan solve     */
} uep_launch_info;
int uep_get_launch_info(const uep_ctx* ctx, uep_launch_info* out);

#ifdef __cplusplus
}
#endif
#endif /* UEP_H_ */
