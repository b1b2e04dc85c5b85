// uf_attn_sm100.cu — step a5, the hot kernel: block-sparse online-softmax attention for B = d = 128
// on sm_100a (KEPT = SINK u TOPK u CUR, R-13/R-14/R-15).
//
// One persistent CTA per SM walks work items (head h, query-block pair p) in head-major order so
// that one head's K/V (25-66 MB) stays L2-resident while it is being used.  A CTA holds two 128-row
// query tiles (blocks 2p, 2p+1) and ping-pongs them on the tensor pipe:
//
//   warp 8   TMA producer : Q tiles once per item; per key block one K tile and one V tile
//                           (128 x 128 bf16, two 64-column boxes, 128-byte swizzle) into smem rings
//   warp 9   MMA issuer   : S_t = Q_t K^T  (tcgen05.mma, SS, M=N=K=128) into TMEM,
//                           O_t += P_t V   (tcgen05.mma, A = P_t from TMEM, B = V tile MN-major)
//   warps 0-3 / 4-7       : softmax of tile 0 / tile 1, one thread per query row: tcgen05.ld the
//                           S row, running max (lazy rescale of O_t in TMEM only when the max grew
//                           by more than 2^8), exp2, row sum, bf16 P back to TMEM over S_t's columns
//   epilogue (same warps) : O_t / l -> bf16 -> swizzled smem (the Q_t buffer) -> TMA store
//
// TMEM (512 columns): S_0 [0,128)  S_1 [128,256)  O_0 [256,384)  O_1 [384,512); P_t aliases the
// first 64 columns of S_t (tensor-pipe ops run in issue order, so S_t(next) is issued after
// O_t += P_t V(prev) and may overwrite it).
//
// Key blocks of an item: first the merged TOPK union of the pair (per entry a 2-bit mask says which
// tile attends it), then SINK, then CUR (both tiles).  All K/V come from the ctx cache.
#include "uf_internal.h"

#include <cstdio>
#include <cstdlib>

namespace {

constexpr int kNK = 3;                 // K ring stages
constexpr int kNV = 2;                 // V ring stages
constexpr int kTile = 128 * 128 * 2;   // bytes of one 128 x 128 bf16 tile
constexpr int kHalf = kTile / 2;       // one 64-column box
constexpr int kThreads = 384;
constexpr float kRescaleThreshold = 8.0f;   // log2 units
#ifdef UF_ARRIVE_ALL
constexpr uint32_t kPArrivals = 128;        // every softmax thread arrives on P_FULL
#else
constexpr uint32_t kPArrivals = 4;          // one elected lane per softmax warp arrives on P_FULL
#endif

// smem carve-up (offsets from a 1024-aligned base)
constexpr int kOffQ = 0;                          // 2 tiles
constexpr int kOffK = kOffQ + 2 * kTile;
constexpr int kOffV = kOffK + kNK * kTile;
constexpr int kOffBar = kOffV + kNV * kTile;
constexpr int kNumBars = 4 + 2 * kNK + 2 * kNV + 6;
constexpr int kOffTmemPtr = kOffBar + kNumBars * 8;
constexpr int kSmemBytes = kOffTmemPtr + 16 + 1024;   // + alignment slack

enum Bar {
  Q_FULL0 = 0, Q_FULL1, Q_EMPTY0, Q_EMPTY1,
  K_FULL0 = 4, K_EMPTY0 = K_FULL0 + kNK,
  V_FULL0 = K_EMPTY0 + kNK, V_EMPTY0 = V_FULL0 + kNV,
  S_FULL0 = V_EMPTY0 + kNV, S_FULL1, P_FULL0, P_FULL1, O_FULL0, O_FULL1
};
static_assert(O_FULL1 + 1 == kNumBars, "barrier count");

// ---- PTX wrappers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t"
      "}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(map), "r"(src), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_store_commit_and_wait_read() {
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void tma_store_wait_all() {
  asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
      "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}

#define UF_TMEM_LD32(taddr, a, o)                                                                              \
  asm volatile(                                                                                                \
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                                                \
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "                                \
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"                \
      : "=r"(a[o + 0]), "=r"(a[o + 1]), "=r"(a[o + 2]), "=r"(a[o + 3]), "=r"(a[o + 4]), "=r"(a[o + 5]),        \
        "=r"(a[o + 6]), "=r"(a[o + 7]), "=r"(a[o + 8]), "=r"(a[o + 9]), "=r"(a[o + 10]), "=r"(a[o + 11]),      \
        "=r"(a[o + 12]), "=r"(a[o + 13]), "=r"(a[o + 14]), "=r"(a[o + 15]), "=r"(a[o + 16]), "=r"(a[o + 17]),  \
        "=r"(a[o + 18]), "=r"(a[o + 19]), "=r"(a[o + 20]), "=r"(a[o + 21]), "=r"(a[o + 22]), "=r"(a[o + 23]),  \
        "=r"(a[o + 24]), "=r"(a[o + 25]), "=r"(a[o + 26]), "=r"(a[o + 27]), "=r"(a[o + 28]), "=r"(a[o + 29]),  \
        "=r"(a[o + 30]), "=r"(a[o + 31])                                                                       \
      : "r"(taddr))

#define UF_TMEM_ST32(taddr, a, o)                                                                              \
  asm volatile(                                                                                                \
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "                                                          \
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "                               \
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"                       \
      ::"r"(taddr), "r"(a[o + 0]), "r"(a[o + 1]), "r"(a[o + 2]), "r"(a[o + 3]), "r"(a[o + 4]), "r"(a[o + 5]),  \
        "r"(a[o + 6]), "r"(a[o + 7]), "r"(a[o + 8]), "r"(a[o + 9]), "r"(a[o + 10]), "r"(a[o + 11]),            \
        "r"(a[o + 12]), "r"(a[o + 13]), "r"(a[o + 14]), "r"(a[o + 15]), "r"(a[o + 16]), "r"(a[o + 17]),        \
        "r"(a[o + 18]), "r"(a[o + 19]), "r"(a[o + 20]), "r"(a[o + 21]), "r"(a[o + 22]), "r"(a[o + 23]),        \
        "r"(a[o + 24]), "r"(a[o + 25]), "r"(a[o + 26]), "r"(a[o + 27]), "r"(a[o + 28]), "r"(a[o + 29]),        \
        "r"(a[o + 30]), "r"(a[o + 31])                                                                         \
      : "memory")

// One lane of a converged warp (the same one every time).  tcgen05.mma / tcgen05.commit / TMA take their
// operands from uniform registers: issued under elect.sync from warp-uniform control flow, ptxas emits them
// straight-line; issued from an `if (lane == 0)` region it wraps EACH one in an ELECT/R2UR/BRA loop
// (~13 instructions, ~70 cycles per MMA: slower than the 64-cycle MMA itself).
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "elect.sync _|p, 0xffffffff;\n\t"
      "selp.b32 %0, 1, 0, p;\n\t"
      "}" : "=r"(pred));
  return pred != 0;
}
// a loaded value every lane holds anyway, made provably warp-uniform for the compiler
__device__ __forceinline__ int32_t uniform_i32(int32_t v) { return __shfl_sync(0xffffffffu, v, 0); }

__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
  float y;
#ifdef UF_DBG_NOMUFU
  y = x * 0.5f;
#else
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
#endif
  return y;
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// ---- packed fp32x2 arithmetic (FFMA2 / FADD2: two lanes per issue slot) and 3-input max (FMNMX3) ----
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t add2_rm(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rm.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t sub2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ float max3(float a, float b, float c) {
  float d;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}

// The MUFU (16 ex2 / cycle / SM) needs as many cycles per 128 x 128 tile as the tensor pipe needs for
// its two MMAs, so a share of the exponentials is computed on the FMA pipe instead: kEmuPairs of every
// 8 column pairs.  2^x = 2^floor(x) * 2^frac(x): floor via the round-down magic-number add (the integer
// lands in the low mantissa bits), 2^frac by a degree-3 minimax polynomial on [0,1) (max relative error
// 7.5e-5, far below the bf16 rounding of P), the exponent added into the float's bits by one LEA.
// Valid for -126 <= x (clamped: the polynomial can return 1 - 7.5e-5, exponent field 126) and x <= 8 (guaranteed by the lazy-rescale invariant).
#ifndef UF_EMU_PAIRS
#define UF_EMU_PAIRS 3
#endif
constexpr int kEmuPairs = UF_EMU_PAIRS;
__device__ __forceinline__ constexpr bool pair_emulated(int j) { return ((j & 7) * kEmuPairs) % 8 < kEmuPairs; }

__device__ __forceinline__ uint64_t ex2_pair(uint64_t x, bool emulate) {
  float x0, x1;
  unpack2(x, x0, x1);
  if (!emulate) return pack2(ex2(x0), ex2(x1));
  const uint64_t magic = pack2(12582912.0f, 12582912.0f);            // 2^23 + 2^22
  x = pack2(fmaxf(x0, -126.0f), fmaxf(x1, -126.0f));
  const uint64_t r = add2_rm(x, magic);
  const uint64_t fr = sub2(x, sub2(r, magic));
  uint64_t p = fma2(fr, pack2(0.07802452147006989f, 0.07802452147006989f), pack2(0.22606715559959412f, 0.22606715559959412f));
  p = fma2(p, fr, pack2(0.6958335638046265f, 0.6958335638046265f));
  p = fma2(p, fr, pack2(0.9999251961708069f, 0.9999251961708069f));
  float p0, p1, r0, r1;
  unpack2(p, p0, p1);
  unpack2(r, r0, r1);
  p0 = __int_as_float((__float_as_int(r0) << 23) + __float_as_int(p0));
  p1 = __int_as_float((__float_as_int(r1) << 23) + __float_as_int(p1));
  return pack2(p0, p1);
}

// One softmax pass over a loaded S row (128 logits in s[]): p = 2^(s*sl2 - m) into bf16 pairs pk[],
// returns the fp32 row sum; with kWithMax also the raw row max (computed beside the exponentials, not
// before them: the running max m used here is the one from the previous key blocks).
template <bool kWithMax>
__device__ __forceinline__ float exp_pass(const uint32_t (&s)[128], uint32_t (&pk)[64], float m, float sl2, float& rowmax) {
  const uint64_t nm2 = pack2(-m, -m), sl22 = pack2(sl2, sl2);
  uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
  float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
  for (int c = 0; c < 128; c += 8) {
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
      const int j = (c + u) >> 1;
      const uint64_t x = fma2(pack2(__uint_as_float(s[c + u]), __uint_as_float(s[c + u + 1])), sl22, nm2);
      const uint64_t p = ex2_pair(x, pair_emulated(j));
      if (j & 1) acc1 = add2(acc1, p); else acc0 = add2(acc0, p);
      float p0, p1;
      unpack2(p, p0, p1);
      pk[j] = pack_bf16x2(p0, p1);
    }
    if (kWithMax) {
      mx0 = max3(mx0, __uint_as_float(s[c + 0]), __uint_as_float(s[c + 1]));
      mx1 = max3(mx1, __uint_as_float(s[c + 2]), __uint_as_float(s[c + 3]));
      mx2 = max3(mx2, __uint_as_float(s[c + 4]), __uint_as_float(s[c + 5]));
      mx3 = max3(mx3, __uint_as_float(s[c + 6]), __uint_as_float(s[c + 7]));
    }
  }
  if (kWithMax) rowmax = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
  float a0, a1, b0, b1;
  unpack2(acc0, a0, a1);
  unpack2(acc1, b0, b1);
  return (a0 + a1) + (b0 + b1);
}

__device__ __forceinline__ float max_pass(const uint32_t (&s)[128]) {
  float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
  for (int c = 0; c < 128; c += 8) {
    mx0 = max3(mx0, __uint_as_float(s[c + 0]), __uint_as_float(s[c + 1]));
    mx1 = max3(mx1, __uint_as_float(s[c + 2]), __uint_as_float(s[c + 3]));
    mx2 = max3(mx2, __uint_as_float(s[c + 4]), __uint_as_float(s[c + 5]));
    mx3 = max3(mx3, __uint_as_float(s[c + 6]), __uint_as_float(s[c + 7]));
  }
  return fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
}

// shared-memory matrix descriptor, 128-byte swizzle
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
         (1ull << 46) | (2ull << 61);
}

// instruction descriptor kind::f16: D fp32, A/B bf16, M = N = 128; B MN-major for P V
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescQK | (1u << 16);

#ifdef UF_DBG_TRACE
// debug only: clock64 timestamps of CTA 0's first kTraceSteps steps; roles: 0 = MMA thread, 1 = softmax tile 0, 2 = softmax tile 1
constexpr int kTraceSteps = 600;
__device__ long long uf_trace[3][kTraceSteps][8];
#define UF_TR(role, step, slot) do { if (blockIdx.x == 0 && (step) < kTraceSteps) uf_trace[role][step][slot] = clock64(); } while (0)
#else
#define UF_TR(role, step, slot) do { } while (0)
#endif

struct AttnParams {
  const int32_t* sel_pair;   // [H][NP][2*kcap]
  const int32_t* pair_cnt;   // [H][NP]
  float* lse;                // [H][ntok] or null
  int H, NP, kcap, np_cur;
  int ntok, nqb;
  int n_sink, sink_ntok;
  int cur_phys0;
  float sl2;                 // softmax scale * log2(e)
};

struct Item {
  int h, p, n_u, n_steps, full_mask;
  const int32_t* ulist;
};

template <bool kUniform = false>
__device__ __forceinline__ Item get_item(const AttnParams& a, int it) {
  Item x;
  x.h = it / a.np_cur;
  x.p = it % a.np_cur;
  const int64_t pi = (int64_t)x.h * a.NP + x.p;
  x.n_u = kUniform ? uniform_i32(a.pair_cnt[pi]) : a.pair_cnt[pi];
  x.ulist = a.sel_pair + pi * 2 * a.kcap;
  x.n_steps = x.n_u + a.n_sink + a.nqb;
  x.full_mask = (2 * x.p + 1 < a.nqb) ? 3 : 1;
  return x;
}

template <bool kUniform = false>
__device__ __forceinline__ int32_t get_entry(const AttnParams& a, const Item& x, int st) {
  if (st < x.n_u) return kUniform ? uniform_i32(__ldg(x.ulist + st)) : __ldg(x.ulist + st);
  st -= x.n_u;
  if (st < a.n_sink) return uf_entry_pack(st, min(128, a.sink_ntok - st * 128), x.full_mask);
  st -= a.n_sink;
  return uf_entry_pack(a.cur_phys0 + st, min(128, a.ntok - st * 128), x.full_mask);
}

__global__ void __launch_bounds__(kThreads, 1)
uf_attn_sm100_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_o,
                     const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                     const AttnParams a) {
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + kOffBar;
  volatile uint32_t* tmem_ptr_smem = reinterpret_cast<volatile uint32_t*>(base_ptr + kOffTmemPtr);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_items = a.H * a.np_cur;

  if (warp == 8 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_o));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_k));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_v));
  }
  if (warp == 9 && lane == 0) {
    for (int i = 0; i < kNumBars; ++i) {
      const bool softmax_arrives = (i == P_FULL0 || i == P_FULL1);
      mbar_init(bars + i * 8, softmax_arrives ? kPArrivals : 1u);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  if (warp == 10) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32((const void*)tmem_ptr_smem)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_smem;
#ifdef UF_DBG_CLOCK
  unsigned long long dbg_c0 = 0, dbg_t0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    dbg_c0 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(dbg_t0));
  }
#endif

  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
    if (warp == 8) {
      // ================================ TMA producer ================================
      // (whole warp runs the control flow; the elected lane issues expect_tx + TMA)
      uint32_t kcount = 0, vcount = 0, qn[2] = {0, 0};
      for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item x = get_item<true>(a, it);
        for (int t = 0; t < 2; ++t) {
          if (!(x.full_mask & (1 << t))) continue;
          const uint32_t bq = bars + (Q_FULL0 + t) * 8;
          mbar_wait(bars + (Q_EMPTY0 + t) * 8, (qn[t] & 1) ^ 1);
          const int row0 = (2 * x.p + t) * 128;
          if (elect_one()) {
            mbar_expect_tx(bq, kTile);
            tma_load_3d(base + kOffQ + t * kTile, &tm_q, bq, 0, row0, x.h);
            tma_load_3d(base + kOffQ + t * kTile + kHalf, &tm_q, bq, 64, row0, x.h);
          }
          ++qn[t];
        }
        int32_t e = get_entry<true>(a, x, 0);
        for (int st = 0; st < x.n_steps; ++st) {
          const int32_t en = (st + 1 < x.n_steps) ? get_entry<true>(a, x, st + 1) : 0;
          const int row = uf_entry_phys(e) * 128;
          {
            const uint32_t s = kcount % kNK, n = kcount / kNK;
            const uint32_t bf = bars + (K_FULL0 + s) * 8;
            mbar_wait(bars + (K_EMPTY0 + s) * 8, (n & 1) ^ 1);
#ifdef UF_DBG_NOTMA
            if (kcount >= kNK) { if (elect_one()) mbar_arrive(bf); } else
#endif
            if (elect_one()) {
            mbar_expect_tx(bf, kTile);
            tma_load_3d(base + kOffK + s * kTile, &tm_k, bf, 0, row, x.h);
            tma_load_3d(base + kOffK + s * kTile + kHalf, &tm_k, bf, 64, row, x.h);
            }
            ++kcount;
          }
          {
            const uint32_t s = vcount % kNV, n = vcount / kNV;
            const uint32_t bf = bars + (V_FULL0 + s) * 8;
            mbar_wait(bars + (V_EMPTY0 + s) * 8, (n & 1) ^ 1);
#ifdef UF_DBG_NOTMA
            if (vcount >= kNV) { if (elect_one()) mbar_arrive(bf); } else
#endif
            if (elect_one()) {
            mbar_expect_tx(bf, kTile);
            tma_load_3d(base + kOffV + s * kTile, &tm_v, bf, 0, row, x.h);
            tma_load_3d(base + kOffV + s * kTile + kHalf, &tm_v, bf, 64, row, x.h);
            }
            ++vcount;
          }
          e = en;
        }
      }
    } else if (warp == 9) {
      // ================================ MMA issuer ==================================
      // (whole warp runs the control flow and the barrier waits; the elected lane issues MMAs and commits)
      uint32_t kcount = 0, vcount = 0, qn[2] = {0, 0}, pn[2] = {0, 0};
      static_assert(kNV == 2, "vrem0/vrem1 below assume a 2-stage V ring");
      int vrem0 = 0, vrem1 = 0;                      // tiles that still have to consume V stage 0 / 1
      for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item x = get_item<true>(a, it);
        bool pend[2] = {false, false};
        uint32_t pend_vs[2] = {0, 0}, pend_vpar[2] = {0, 0};
        bool first_pv[2] = {true, true};
        for (int t = 0; t < 2; ++t)
          if (x.full_mask & (1 << t)) { mbar_wait(bars + (Q_FULL0 + t) * 8, qn[t] & 1); ++qn[t]; }

        auto do_pv = [&](int t) {
          UF_TR(0, (int)kcount, t * 2);
          mbar_wait(bars + (P_FULL0 + t) * 8, pn[t] & 1); ++pn[t];
          UF_TR(0, (int)kcount, t * 2 + 1);
          const uint32_t vs = pend_vs[t];
          mbar_wait(bars + (V_FULL0 + vs) * 8, pend_vpar[t]);
          tc_fence_after();
          const uint32_t vaddr = base + kOffV + vs * kTile;
          const uint32_t d_tmem = tmem + 256 + t * 128;
          const uint32_t p_tmem = tmem + t * 128;
          const int left = (vs == 0) ? --vrem0 : --vrem1;
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              // B = V tile, MN-major: 8-key groups 1024 B apart (SBO), the two 64-column halves 16 KB apart (LBO)
              const uint64_t bd = make_desc(vaddr + k * 2048, kHalf, 1024);
#ifndef UF_DBG_NOPV
              mma_ts(d_tmem, p_tmem + k * 8, bd, kIdescPV, (first_pv[t] && k == 0) ? 0u : 1u);
#endif
            }
            if (left == 0) tc_commit(bars + (V_EMPTY0 + vs) * 8);
          }
          __syncwarp();
          first_pv[t] = false;
          pend[t] = false;
        };

        int32_t e = get_entry<true>(a, x, 0);
        for (int st = 0; st < x.n_steps; ++st) {
          const int32_t en = (st + 1 < x.n_steps) ? get_entry<true>(a, x, st + 1) : 0;
          const int m = uf_entry_mask(e);
          const uint32_t ks = kcount % kNK, kpar = (kcount / kNK) & 1;
          const uint32_t vs = vcount % kNV, vpar = (vcount / kNV) & 1;
          UF_TR(0, (int)kcount, 6);
          mbar_wait(bars + (K_FULL0 + ks) * 8, kpar);
          UF_TR(0, (int)kcount, 7);
          tc_fence_after();
          UF_TR(0, (int)kcount, 4);
          const uint32_t kaddr = base + kOffK + ks * kTile;
          int users = 0;
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            if (!(m & (1 << t))) continue;
            if (pend[t]) do_pv(t);
            const uint32_t qaddr = base + kOffQ + t * kTile;
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                // K-major operands: 8-row groups 1024 B apart (SBO); 16 elements = 32 B along K, second half +16 KB
                const uint32_t koff = (k & 3) * 32 + (k >> 2) * kHalf;
#ifndef UF_DBG_NOQK
                mma_ss(tmem + t * 128, make_desc(qaddr + koff, 16, 1024), make_desc(kaddr + koff, 16, 1024), kIdescQK,
                       k == 0 ? 0u : 1u);
#endif
              }
              tc_commit(bars + (S_FULL0 + t) * 8);
            }
            __syncwarp();
            pend[t] = true; pend_vs[t] = vs; pend_vpar[t] = vpar;
            ++users;
          }
          if (elect_one()) tc_commit(bars + (K_EMPTY0 + ks) * 8);
          __syncwarp();
          UF_TR(0, (int)kcount, 5);
          if (vs == 0) vrem0 = users; else vrem1 = users;
          ++kcount; ++vcount;
#pragma unroll
          for (int t = 0; t < 2; ++t)
            if (!(m & (1 << t)) && pend[t]) do_pv(t);      // keep V stages flowing (no deadlock)
          e = en;
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (pend[t]) do_pv(t);
          if (x.full_mask & (1 << t)) {
            if (elect_one()) tc_commit(bars + (O_FULL0 + t) * 8);
            __syncwarp();
          }
        }
      }
    }
  } else {
    // ================================== softmax + epilogue ==================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    const int t = warp >> 2;                           // tile
    const int wq = warp & 3;                           // TMEM lane quarter
    const int row = wq * 32 + lane;                    // row in the tile == TMEM lane
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    const uint32_t s_tmem = tmem + lane_addr + t * 128;
    const uint32_t o_tmem = tmem + lane_addr + 256 + t * 128;
    const uint32_t b_sfull = bars + (S_FULL0 + t) * 8;
    const uint32_t b_pfull = bars + (P_FULL0 + t) * 8;
    const uint32_t b_ofull = bars + (O_FULL0 + t) * 8;
    const uint32_t b_qempty = bars + (Q_EMPTY0 + t) * 8;
    unsigned char* stage = base_ptr + kOffQ + t * kTile;
    uint32_t sn = 0, on = 0;
    for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
      const Item x = get_item(a, it);
      if (!(x.full_mask & (1 << t))) continue;
      float m = -INFINITY, l = 0.f;
      bool first = true;
      int32_t e = get_entry(a, x, 0);
      for (int st = 0; st < x.n_steps; ++st) {
        const int32_t en = (st + 1 < x.n_steps) ? get_entry(a, x, st + 1) : 0;
        const int32_t ecur = e;
        e = en;
        if (!(uf_entry_mask(ecur) & (1 << t))) continue;
        const int nvalid = uf_entry_nvalid(ecur);
        if (wq == 0 && lane == 0) UF_TR(1 + t, (int)sn, 0);
        mbar_wait(b_sfull, sn & 1); ++sn;
        tc_fence_after();
        if (wq == 0 && lane == 0) UF_TR(1 + t, (int)sn - 1, 1);
#ifdef UF_DBG_NOSOFTMAX
        l = 1.f;
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(b_pfull);
        if (wq == 0 && lane == 0) UF_TR(1 + t, (int)sn - 1, 2);
        continue;
#endif
        uint32_t s[128];
        uint32_t pk[64];
        auto load_s = [&]() {
          UF_TMEM_LD32(s_tmem + 0, s, 0);
          UF_TMEM_LD32(s_tmem + 32, s, 32);
          UF_TMEM_LD32(s_tmem + 64, s, 64);
          UF_TMEM_LD32(s_tmem + 96, s, 96);
          tmem_wait_ld();
          if (nvalid < 128) {
#pragma unroll
            for (int c = 0; c < 128; ++c)
              if (c >= nvalid) s[c] = 0xff800000u;     // -inf: ragged key block (R-3)
          }
        };
        load_s();
        float lsum, rowmax = 0.f;
#ifdef UF_DBG_NOEXP
        lsum = 1.f;
#pragma unroll
        for (int c = 0; c < 64; ++c) pk[c] = s[c] ^ s[c + 64];
#else
        if (first) {
          m = max_pass(s) * a.sl2;
          first = false;
          lsum = exp_pass<false>(s, pk, m, a.sl2, rowmax);
        } else {
          // Exponentials against the running max of the EARLIER blocks, the row max of this block
          // computed beside them: the max -> exp dependency leaves the critical path.  Valid while
          // the new max exceeds m by at most 2^8 (the lazy-rescale invariant); otherwise redo.
          lsum = exp_pass<true>(s, pk, m, a.sl2, rowmax);
          const float m_new = fmaxf(m, rowmax * a.sl2);
          const bool need = (m_new - m) > kRescaleThreshold;
          if (__any_sync(0xffffffffu, need)) {
            // O_t is quiescent here: S_t's commit covers the earlier O_t += P_t V
            const float f = need ? ex2(m - m_new) : 1.0f;
            if (need) { m = m_new; l *= f; }
#pragma unroll
            for (int cc = 0; cc < 128; cc += 32) {
              uint32_t ov[32];
              UF_TMEM_LD32(o_tmem + cc, ov, 0);
              tmem_wait_ld();
#pragma unroll
              for (int c = 0; c < 32; ++c) ov[c] = __float_as_uint(__uint_as_float(ov[c]) * f);
              UF_TMEM_ST32(o_tmem + cc, ov, 0);
            }
            load_s();
            lsum = exp_pass<false>(s, pk, m, a.sl2, rowmax);
          }
        }
#endif
        l += lsum;
        UF_TMEM_ST32(s_tmem + 0, pk, 0);
        UF_TMEM_ST32(s_tmem + 32, pk, 32);
        tmem_wait_st();
        tc_fence_before();
#ifdef UF_ARRIVE_ALL
        mbar_arrive(b_pfull);
#else
        __syncwarp();
        if (lane == 0) mbar_arrive(b_pfull);
#endif
        if (wq == 0 && lane == 0) UF_TR(1 + t, (int)sn - 1, 2);
      }
      // ---- epilogue: O_t / l -> bf16 -> swizzled staging (Q_t buffer) -> TMA store ----
      mbar_wait(b_ofull, on & 1); ++on;
      tc_fence_after();
      const float inv = 1.0f / l;
#pragma unroll
      for (int cc = 0; cc < 128; cc += 32) {
        uint32_t ov[32];
        UF_TMEM_LD32(o_tmem + cc, ov, 0);
        tmem_wait_ld();
        unsigned char* half_base = stage + (cc >> 6) * kHalf + row * 128;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint4 w;
          w.x = pack_bf16x2(__uint_as_float(ov[8 * j + 0]) * inv, __uint_as_float(ov[8 * j + 1]) * inv);
          w.y = pack_bf16x2(__uint_as_float(ov[8 * j + 2]) * inv, __uint_as_float(ov[8 * j + 3]) * inv);
          w.z = pack_bf16x2(__uint_as_float(ov[8 * j + 4]) * inv, __uint_as_float(ov[8 * j + 5]) * inv);
          w.w = pack_bf16x2(__uint_as_float(ov[8 * j + 6]) * inv, __uint_as_float(ov[8 * j + 7]) * inv);
          const int chunk = ((cc & 63) >> 3) + j;                  // 16-byte chunk within the 128-byte row
          *reinterpret_cast<uint4*>(half_base + ((chunk ^ (row & 7)) << 4)) = w;
        }
      }
      tc_fence_before();
      fence_proxy_async();
      asm volatile("bar.sync %0, 128;" ::"r"(1 + t) : "memory");
      const int row0 = (2 * x.p + t) * 128;
      if (wq == 0 && lane == 0) {
        const uint32_t src = base + kOffQ + t * kTile;
        tma_store_3d(&tm_o, src, 0, row0, x.h);
        tma_store_3d(&tm_o, src + kHalf, 64, row0, x.h);
        tma_store_commit_and_wait_read();
        mbar_arrive(b_qempty);
      }
      if (a.lse != nullptr && row0 + row < a.ntok)
        a.lse[(int64_t)x.h * a.ntok + row0 + row] = (m + log2f(l)) * 0.6931471805599453f;
    }
    if (wq == 0 && lane == 0) tma_store_wait_all();
  }

  tc_fence_before();
  __syncthreads();
#ifdef UF_DBG_CLOCK
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long c1 = clock64(), t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    printf("UFCLK cycles %llu ns %llu MHz %.1f\n", c1 - dbg_c0, t1 - dbg_t0, 1e3 * (double)(c1 - dbg_c0) / (double)(t1 - dbg_t0));
  }
#endif
  if (warp == 10) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = nullptr;
  if (fn) return fn;
  void* p = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
      qres != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<PFN_encodeTiled>(p);
  return fn;
}

// bf16 tensor [rows, H, 128] with element strides (row_stride, head_stride, 1); box = 64 x 128 x 1
bool encode_map(CUtensorMap* m, const void* ptr, uint64_t rows, uint64_t H, uint64_t row_stride, uint64_t head_stride) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[3] = {128, rows, H};
  const cuuint64_t strides[2] = {row_stride * 2, head_stride * 2};
  const cuuint32_t box[3] = {64, 128, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

int uf_sm100_make_cache_maps(uf_ctx* c) {
  const uint64_t rows = (uint64_t)c->P * 128;
  if (!encode_map(&c->tm_k, c->kc, rows, c->cfg.n_heads, 128, rows * 128) ||
      !encode_map(&c->tm_v, c->vc, rows, c->cfg.n_heads, 128, rows * 128)) {
    c->err = "cuTensorMapEncodeTiled failed for the K/V cache";
    return UF_ERR_CUDA;
  }
  cudaError_t e = cudaFuncSetAttribute(uf_attn_sm100_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) {
    c->err = std::string("cudaFuncSetAttribute(smem): ") + cudaGetErrorString(e);
    return UF_ERR_CUDA;
  }
  c->tm_ok = true;
  return UF_OK;
}

int uf_launch_attn_sm100(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, __nv_bfloat16* o, float* lse,
                         int64_t tok_stride, int64_t head_stride, float scale, cudaStream_t s) {
  CUtensorMap tm_q, tm_o;
  if (!encode_map(&tm_q, q, v.cur_ntok, v.H, tok_stride, head_stride) ||
      !encode_map(&tm_o, o, v.cur_ntok, v.H, tok_stride, head_stride)) {
    c->err = "cuTensorMapEncodeTiled failed for Q/O (check strides and alignment)";
    return UF_ERR_INVALID_ARG;
  }
  AttnParams a;
  a.sel_pair = c->sel_pair; a.pair_cnt = c->pair_cnt; a.lse = lse;
  a.H = v.H; a.NP = (v.BPC + 1) / 2; a.kcap = c->kcap;
  a.ntok = v.cur_ntok; a.nqb = uf_ceil_div(v.cur_ntok, 128); a.np_cur = (a.nqb + 1) / 2;
  a.n_sink = v.n_sink_blocks; a.sink_ntok = v.sink_ntok;
  a.cur_phys0 = v.S + v.cur_slot * v.BPC;
  a.sl2 = scale * 1.4426950408889634f;
  const int n_items = a.H * a.np_cur;
  const int grid = n_items < c->sm_count ? n_items : c->sm_count;
  uf_attn_sm100_kernel<<<grid, kThreads, kSmemBytes, s>>>(tm_q, tm_o, c->tm_k, c->tm_v, a);
  c->launches += 1;
#ifdef UF_DBG_TRACE
  if (const char* path = getenv("UF_TRACE_PATH")) {
    cudaDeviceSynchronize();
    static long long host[3][kTraceSteps][8];
    cudaMemcpyFromSymbol(host, uf_trace, sizeof(host));
    if (FILE* f = fopen(path, "wb")) { fwrite(host, 1, sizeof(host), f); fclose(f); }
  }
#endif
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    c->err = std::string("uf_attn_sm100_kernel launch: ") + cudaGetErrorString(e);
    return UF_ERR_CUDA;
  }
  return UF_OK;
}
