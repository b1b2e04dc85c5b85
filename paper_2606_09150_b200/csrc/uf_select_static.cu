// uf_select_static.cu — uf_select_blocks_static (include/uf_static.h): steps a2-a4 (block-mean pooling P:90, scores
// Eq. 4, exact top-k with ties to the lower index) for hosts that may not allocate device memory.  The pooled
// Q / K tables, which uf_select_blocks keeps in cudaMalloc'ed ctx memory, live here in a fixed `static __device__`
// array.  This file is self-contained: it shares no kernel and no state with uf_select.cu, and nothing in it calls
// cudaMalloc, cudaFree, cudaFuncSetAttribute or any allocating library routine.
//
// Arithmetic (same as uf_select.cu, R-3/R-4): block sums in fp64 (exact for <= 128 bf16 values, hence
// order-free), mean = sum / valid rows, score = products and sums rounded separately in channel order, then one
// division by sqrt(d); -0.0 is normalised to +0.0 before ranking.
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "uf.h"
#include "uf_static.h"

// The scratch array.  In HOST code this name is only a handle for the runtime's symbol table, not an address a
// kernel can use: the device address is looked up per GPU with cudaGetSymbolAddress (scratch_on_device below) and
// handed to the kernels as an ordinary pointer.
static __device__ __align__(256) unsigned char uf_static_scratch[UF_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

// Device address of uf_static_scratch on each GPU, looked up once per GPU with that GPU current.
std::mutex g_mu;
unsigned char* g_scratch[kMaxDevices] = {};

cudaError_t scratch_on_device(int device, unsigned char** out) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_scratch[device] == nullptr) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, uf_static_scratch);     // the caller made `device` current
    if (e != cudaSuccess) return e;
    g_scratch[device] = static_cast<unsigned char*>(p);
  }
  *out = g_scratch[device];
  return cudaSuccess;
}

__device__ __forceinline__ uint4 ld_once(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// ---- pooling: grid (nqb + nkb, H).  CTAs [0, nqb) pool Q into qbar [H][nqb][D]; CTAs [nqb, nqb + nkb) pool K
// into kbar [H][D][nkb] (transposed: the scoring loop reads one channel of consecutive key blocks per warp).
template <int D>
__global__ void __launch_bounds__(kThreads)
uf_static_pool_kernel(const __nv_bfloat16* __restrict__ q, int64_t q_ts, int64_t q_hs, int nq,
                      const __nv_bfloat16* __restrict__ k, int64_t k_ts, int64_t k_hs, int nk,
                      int B, int nqb, int nkb, double* __restrict__ qbar, double* __restrict__ kbar) {
  constexpr int VPR = D / 8;                 // 16-byte vectors per row
  constexpr int RPP = kThreads / VPR;        // rows per pass
  __shared__ double red[RPP][D + 2];
  const bool is_q = (int)blockIdx.x < nqb;
  const int b = is_q ? blockIdx.x : blockIdx.x - nqb;
  const int h = blockIdx.y;
  const __nv_bfloat16* src = is_q ? q : k;
  const int64_t ts = is_q ? q_ts : k_ts, hs = is_q ? q_hs : k_hs;
  const int nvalid = min(B, (is_q ? nq : nk) - b * B);
  const int vc = threadIdx.x % VPR, rg = threadIdx.x / VPR;
  double acc[8];
#pragma unroll
  for (int t = 0; t < 8; ++t) acc[t] = 0.0;
  for (int r = rg; r < nvalid; r += RPP) {
    const uint4 u = ld_once(reinterpret_cast<const uint4*>(src + (int64_t)(b * B + r) * ts + (int64_t)h * hs + vc * 8));
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      acc[2 * t]     += (double)__uint_as_float(w[t] << 16);
      acc[2 * t + 1] += (double)__uint_as_float(w[t] & 0xFFFF0000u);
    }
  }
#pragma unroll
  for (int t = 0; t < 8; ++t) red[rg][vc * 8 + t] = acc[t];
  __syncthreads();
  if (threadIdx.x < D) {
    double s = 0.0;
#pragma unroll
    for (int g = 0; g < RPP; ++g) s += red[g][threadIdx.x];
    const double mean = s / (double)nvalid;
    if (is_q) qbar[((int64_t)h * nqb + b) * D + threadIdx.x] = mean;
    else      kbar[((int64_t)h * D + threadIdx.x) * nkb + b] = mean;
  }
}

// order-preserving map double -> uint64 (finite inputs; -0.0 already normalised)
__device__ __forceinline__ unsigned long long sortable(double x) {
  const unsigned long long u = (unsigned long long)__double_as_longlong(x);
  return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}

// ---- scores + top-k: grid (nqb, H), one query block per CTA, its nkb keys ranked in shared memory.
template <int D>
__global__ void __launch_bounds__(kThreads)
uf_static_score_topk_kernel(const double* __restrict__ qbar, const double* __restrict__ kbar, int nqb, int nkb,
                            int k_eff, int32_t* __restrict__ idx_out) {
  __shared__ double qs[D];
  __shared__ unsigned long long key[UF_STATIC_MAX_KEY_BLOCKS];
  const int i = blockIdx.x, h = blockIdx.y, tid = threadIdx.x;
  if (tid < D) qs[tid] = qbar[((int64_t)h * nqb + i) * D + tid];
  __syncthreads();
  const double root = sqrt((double)D);
  for (int j = tid; j < nkb; j += kThreads) {
    const double* kp = kbar + (int64_t)h * D * nkb + j;
    double acc = 0.0;
#pragma unroll 8
    for (int t = 0; t < D; ++t) acc = __dadd_rn(acc, __dmul_rn(qs[t], kp[(int64_t)t * nkb]));
    key[j] = sortable(__ddiv_rn(acc, root) + 0.0);
  }
  __syncthreads();
  // T = the largest value with #{key >= T} >= k', built bit by bit from the top.  Kept: every key > T and, of the
  // keys == T, the first k' - #{key > T} in index order (ties to the lower block index).
  __shared__ int wcnt[kThreads / 32];
  unsigned long long T = 0ull;
  for (int b = 63; b >= 0; --b) {
    const unsigned long long cand = T | (1ull << b);
    int mine = 0;
    for (int j = tid; j < nkb; j += kThreads) mine += (key[j] >= cand);
    mine = __reduce_add_sync(0xffffffffu, mine);
    if ((tid & 31) == 0) wcnt[tid >> 5] = mine;
    __syncthreads();
    int tot = 0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) tot += wcnt[w];
    __syncthreads();                                         // wcnt is rewritten in the next round
    if (tot >= k_eff) T = cand;
  }
  if (tid < 32) {                                            // ordered compaction by one warp: ascending indices
    const int lane = tid;
    int n_gt = 0;
    for (int j = lane; j < nkb; j += 32) n_gt += (key[j] > T);
    n_gt = __reduce_add_sync(0xffffffffu, n_gt);
    const int need_eq = k_eff - n_gt;
    int32_t* row = idx_out + ((int64_t)h * nqb + i) * k_eff;
    int pos0 = 0, eq_seen = 0;
    for (int j0 = 0; j0 < nkb; j0 += 32) {
      const int j = j0 + lane;
      const unsigned long long mine = j < nkb ? key[j] : 0ull;
      const bool gt = j < nkb && mine > T, eq = j < nkb && mine == T;
      const unsigned beq = __ballot_sync(0xffffffffu, eq);
      const bool keep = gt || (eq && eq_seen + __popc(beq & ((1u << lane) - 1u)) < need_eq);
      const unsigned ball = __ballot_sync(0xffffffffu, keep);
      if (keep) row[pos0 + __popc(ball & ((1u << lane) - 1u))] = j;
      pos0 += __popc(ball);
      eq_seen += __popc(beq);
    }
  }
}

int check_tensor(const void* p, int64_t ts, int64_t hs, int d, const char* name) {
  if (!p) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: %s is null", name);
  if (((uintptr_t)p & 15) != 0) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: %s not 16-byte aligned", name);
  if (ts < d || hs < d || (ts % 8) || (hs % 8))
    return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: %s strides must be >= head_dim and multiples of 8 elements", name);
  return UF_OK;
}

}  // namespace

extern "C" const char* uf_static_last_error(void) { return g_err; }

extern "C" int32_t uf_select_blocks_static(int32_t device,
                                           const void* q, int32_t n_q_tokens, int64_t q_tok_stride, int64_t q_head_stride,
                                           const void* k, int32_t n_k_tokens, int64_t k_tok_stride, int64_t k_head_stride,
                                           int32_t n_heads, int32_t head_dim, int32_t block, int32_t topk_count,
                                           int32_t* idx_out, void* stream) {
  // ---- arguments and sizes first: nothing below this block runs for a problem that does not fit ----
  if (device < 0 || device >= kMaxDevices) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: device %d outside 0..%d", device, kMaxDevices - 1);
  if (head_dim != 32 && head_dim != 64 && head_dim != 128) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: head_dim must be 32, 64 or 128");
  if (block < 32 || block > 128 || block % 32) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: block must be 32, 64, 96 or 128");
  if (n_heads < 1 || n_heads > 65535) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: n_heads outside 1..65535");
  if (n_q_tokens < 1 || n_k_tokens < 1) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: n_q_tokens and n_k_tokens must be >= 1");
  if (topk_count < 1) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: topk_count must be >= 1");
  if (!idx_out) return fail(UF_ERR_INVALID_ARG, "uf_select_blocks_static: idx_out is null");
  int rc = check_tensor(q, q_tok_stride, q_head_stride, head_dim, "q");
  if (rc != UF_OK) return rc;
  rc = check_tensor(k, k_tok_stride, k_head_stride, head_dim, "k");
  if (rc != UF_OK) return rc;
  const int64_t nqb = ((int64_t)n_q_tokens + block - 1) / block, nkb = ((int64_t)n_k_tokens + block - 1) / block;
  if (nkb > UF_STATIC_MAX_KEY_BLOCKS)
    return fail(UF_ERR_CAPACITY, "uf_select_blocks_static: %lld key blocks, the limit is %d (UF_STATIC_MAX_KEY_BLOCKS)",
                (long long)nkb, UF_STATIC_MAX_KEY_BLOCKS);
  const int64_t q_bytes = ((8 * (int64_t)n_heads * head_dim * nqb + 255) / 256) * 256;
  const int64_t k_bytes = 8 * (int64_t)n_heads * head_dim * nkb;
  if (q_bytes + k_bytes > (int64_t)UF_STATIC_SCRATCH_BYTES)
    return fail(UF_ERR_CAPACITY, "uf_select_blocks_static: pooled tables need %lld bytes, the static array holds %d "
                "(UF_STATIC_SCRATCH_BYTES); use uf_select_blocks with a ctx for this size",
                (long long)(q_bytes + k_bytes), UF_STATIC_SCRATCH_BYTES);
  if (nqb + nkb > 0x7fffffffLL) return fail(UF_ERR_CAPACITY, "uf_select_blocks_static: too many blocks for one grid");
  const int k_eff = topk_count < nkb ? topk_count : (int)nkb;

  // ---- device: make it current, fetch (first call on this GPU: look up) the array's device address ----
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return fail(UF_ERR_CUDA, "uf_select_blocks_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
  unsigned char* scratch = nullptr;
  e = scratch_on_device(device, &scratch);
  if (e != cudaSuccess) return fail(UF_ERR_CUDA, "uf_select_blocks_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  double* qbar = reinterpret_cast<double*>(scratch);
  double* kbar = reinterpret_cast<double*>(scratch + q_bytes);

  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const __nv_bfloat16* qp = static_cast<const __nv_bfloat16*>(q);
  const __nv_bfloat16* kp = static_cast<const __nv_bfloat16*>(k);
  const dim3 gpool((unsigned)(nqb + nkb), (unsigned)n_heads), gscore((unsigned)nqb, (unsigned)n_heads);
#define UF_STATIC_CASE(DD)                                                                                        \
  case DD:                                                                                                        \
    uf_static_pool_kernel<DD><<<gpool, kThreads, 0, s>>>(qp, q_tok_stride, q_head_stride, n_q_tokens, kp,         \
                                                         k_tok_stride, k_head_stride, n_k_tokens, block,          \
                                                         (int)nqb, (int)nkb, qbar, kbar);                         \
    uf_static_score_topk_kernel<DD><<<gscore, kThreads, 0, s>>>(qbar, kbar, (int)nqb, (int)nkb, k_eff, idx_out);  \
    break;
  switch (head_dim) {
    UF_STATIC_CASE(32)
    UF_STATIC_CASE(64)
    UF_STATIC_CASE(128)
  }
#undef UF_STATIC_CASE
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(UF_ERR_CUDA, "uf_select_blocks_static: kernel launch: %s", cudaGetErrorString(e));
  return UF_OK;
}
