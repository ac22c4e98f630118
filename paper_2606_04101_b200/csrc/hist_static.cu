// hist_static.cu — uep_histogram_static: lambda_e = #{s : topk_ids[s] == e}  (Alg. 1 line 2,
// PAPER.md:250) for callers that cannot allocate: no context, no workspace, no cudaMalloc anywhere
// on the path.  A variant of hist_kernel<true> (hist.cu) whose scratch — the per-CTA count rows —
// lives in a file-scope __device__ array of fixed size instead of the caller's workspace:
//
//   hist_static_kernel   CTA c counts its block of slots in shared memory (same counting scheme as
//                        hist_kernel: 8 rows of counters shared by 4 warps each, 4 x 16-byte loads
//                        in flight per thread) and stores its column sums as row c of the scratch
//   sum_static_kernel    one CTA: expert_count[e] = sum over rows in row order (integer adds)
//
// Every row a call reads was written in full by the same call, so nothing has to start at zero and
// nothing is cleared; the rows keep the last call's values.  ALL calls on a device share the one
// array: two calls that overlap on the GPU (different streams, or one graph replayed concurrently
// with itself) race on it.  The array (kStaticRows x UEP_MAX_E x 4 B = 384 KB) is part of the
// library's image on every GPU that loads it, until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current
// (static_setup below).
#include <mutex>
#include <cstdio>

#include "uep_internal.cuh"

namespace uep {

constexpr int kStaticRows = 192;                              // >= the SM count of the part (148)
constexpr int kStaticThreads = 1024;
constexpr int kStaticShare = 2;                               // log2 of the warps sharing a row of counters
constexpr int kStaticCntRows = (kStaticThreads / 32) >> kStaticShare;
constexpr int kStaticVecs = 4;                                // int4 loads per thread per round
constexpr int kStaticPitch = UEP_MAX_E + 1;                   // the same expert of two rows: different banks
constexpr int kStaticMaxDev = 64;

static __device__ __align__(256) int32_t g_static_rows[kStaticRows * UEP_MAX_E];

__global__ void __launch_bounds__(kStaticThreads, 1)
hist_static_kernel(const int32_t* __restrict__ ids, long long S, int E, int per,
                   int32_t* __restrict__ rows) {
  __shared__ int priv[kStaticCntRows * kStaticPitch];
  const int tid = threadIdx.x, warp = tid >> 5;
  const long long begin = (long long)blockIdx.x * per;
  const int len = (int)min((long long)per, S - begin);                    // > 0 by construction
  const int n_vec = len >> 2;
  const int4* v = reinterpret_cast<const int4*>(ids + begin);             // per % 128 == 0, ids 16-B aligned

  int4 x[kStaticVecs];
#pragma unroll
  for (int u = 0; u < kStaticVecs; ++u) {
    const int i = u * kStaticThreads + tid;
    x[u] = (i < n_vec) ? __ldg(v + i) : make_int4(-1, -1, -1, -1);
  }
  for (int i = tid; i < kStaticCntRows * kStaticPitch; i += kStaticThreads) priv[i] = 0;
  __syncthreads();

  int* row = priv + (warp >> kStaticShare) * kStaticPitch;
  auto count_one = [&](int e) { if ((unsigned)e < (unsigned)E) atomicAdd(&row[e], 1); };   // S14: invalid ids skipped
  for (int vbase = 0; vbase < n_vec; vbase += kStaticThreads * kStaticVecs) {
#pragma unroll
    for (int u = 0; u < kStaticVecs; ++u) {
      count_one(x[u].x); count_one(x[u].y); count_one(x[u].z); count_one(x[u].w);
    }
    const int nb = vbase + kStaticThreads * kStaticVecs;
    if (nb < n_vec) {
#pragma unroll
      for (int u = 0; u < kStaticVecs; ++u) {
        const int i = nb + u * kStaticThreads + tid;
        x[u] = (i < n_vec) ? __ldg(v + i) : make_int4(-1, -1, -1, -1);
      }
    }
  }
  if (tid < (len & 3)) count_one(ids[begin + (n_vec << 2) + tid]);        // ragged tail
  __syncthreads();

  for (int e = tid; e < E; e += kStaticThreads) {
    int s = 0;
#pragma unroll
    for (int w = 0; w < kStaticCntRows; ++w) s += priv[w * kStaticPitch + e];
    rows[(size_t)blockIdx.x * UEP_MAX_E + e] = s;                         // the whole row [0, E), every call
  }
}

__global__ void __launch_bounds__(UEP_MAX_E)
sum_static_kernel(int E, int n_rows, const int32_t* __restrict__ rows, int32_t* __restrict__ expert_count) {
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    int s = 0;
#pragma unroll 8
    for (int r = 0; r < n_rows; ++r) s += __ldcg(rows + (size_t)r * UEP_MAX_E + e);
    expert_count[e] = s;
  }
}

// per device: the scratch's device address and the grid size; filled once, under the mutex
struct StaticDev { int32_t* rows; int n_ctas; bool ready; };
static StaticDev g_static_dev[kStaticMaxDev];
static std::mutex g_static_mu;
static thread_local char g_static_err[256] = "";

// (arguments the text does not name are ignored)
static int static_fail(int rc, const char* fmt, long long a = 0, long long b = 0) {
  std::snprintf(g_static_err, sizeof(g_static_err), fmt, a, b);
  return rc;
}

// Once per device, with that device current: resolve the scratch's address on THIS device.
static int static_setup(StaticDev** out) {
  int dev = -1;
  UEP_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDev)
    return static_fail(UEP_ERR_UNSUPPORTED, "uep_histogram_static: device ordinal %lld outside [0, %lld)", dev, kStaticMaxDev);
  std::lock_guard<std::mutex> lock(g_static_mu);
  StaticDev& d = g_static_dev[dev];
  if (!d.ready) {
    int major = 0, sms = 0;
    UEP_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    UEP_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return static_fail(UEP_ERR_UNSUPPORTED, "uep_histogram_static: compute capability %lld.x, built for sm_100a only", major);
    void* p = nullptr;
    UEP_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_rows));
    if (p == nullptr) return static_fail(UEP_ERR_CUDA, "uep_histogram_static: cudaGetSymbolAddress gave a null address");
    d.rows = static_cast<int32_t*>(p);
    d.n_ctas = sms < 1 ? 1 : (sms > kStaticRows ? kStaticRows : sms);
    d.ready = true;
  }
  *out = &d;
  return UEP_OK;
}

}  // namespace uep

extern "C" {

int uep_histogram_static_setup(void) {
  uep::StaticDev* d = nullptr;
  return uep::static_setup(&d);
}

int uep_histogram_static(const int32_t* topk_ids, long long n_slots, int32_t E, int32_t* expert_count,
                         void* stream) {
  using namespace uep;
  g_static_err[0] = 0;
  if (n_slots < 0) return static_fail(UEP_ERR_INVALID_ARG, "uep_histogram_static: n_slots %lld < 0", n_slots);
  if (n_slots > (long long)UEP_STATIC_MAX_SLOTS)
    return static_fail(UEP_ERR_UNSUPPORTED, "uep_histogram_static: n_slots %lld exceeds UEP_STATIC_MAX_SLOTS %lld", n_slots,
                       (long long)UEP_STATIC_MAX_SLOTS);
  if (E < 1 || E > UEP_MAX_E)
    return static_fail(UEP_ERR_UNSUPPORTED, "uep_histogram_static: E %lld outside [1, UEP_MAX_E = %lld]", E, UEP_MAX_E);
  if (expert_count == nullptr || (n_slots > 0 && topk_ids == nullptr) ||
      (reinterpret_cast<uintptr_t>(topk_ids) & 15) || (reinterpret_cast<uintptr_t>(expert_count) & 15))
    return static_fail(UEP_ERR_INVALID_ARG, "uep_histogram_static: NULL or not 16-byte aligned pointer");
  StaticDev* d = nullptr;
  const int rc = static_setup(&d);
  if (rc != UEP_OK) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // CTA c counts the slots [c * per, (c + 1) * per): whole 128-slot lines, at most one block per SM
  long long per = (n_slots + d->n_ctas - 1) / d->n_ctas;
  per = (per + 127) / 128 * 128;
  const int n_rows = per > 0 ? (int)((n_slots + per - 1) / per) : 0;       // <= n_ctas <= kStaticRows
  if (n_rows > 0) {
    hist_static_kernel<<<n_rows, kStaticThreads, 0, s>>>(topk_ids, n_slots, E, (int)per, d->rows);
    UEP_CUDA_TRY(cudaGetLastError());
  }
  sum_static_kernel<<<1, E < 32 ? 32 : (E + 31) / 32 * 32, 0, s>>>(E, n_rows, d->rows, expert_count);
  UEP_CUDA_TRY(cudaGetLastError());
  return UEP_OK;
}

const char* uep_static_last_error(void) { return uep::g_static_err; }

}  // extern "C"
