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
//   warps 0-7             : softmax of tile 0 and tile 1 in turn, TWO threads per query row (64 keys
//                           each), S read from TMEM in 32-column chunks (next chunk in flight while
//                           this one is processed), bf16 P written back over the thread's own S columns
//   epilogue (same warps) : O_t / l -> bf16 -> swizzled smem (the Q_t buffer) -> TMA store
//
// Warps 8 and 9 run their control flow warp-uniformly and issue TMA / tcgen05.mma / tcgen05.commit
// from the lane elect.sync picks: those instructions take uniform-register operands, and issued from
// an `if (lane == 0)` region ptxas wraps EACH one in an ELECT/R2UR/BRA loop (measured: ~70 cycles per
// MMA, slower than the 64-cycle MMA).  The tensor pipe's command queue is shallow (issue blocks while
// it is full), so whatever the MMA warp executes between two MMA groups is exposed: descriptors are
// a precomputed 32-bit base plus a constant, stage counters are incremental, entries are prefetched.
//
// Softmax (R-20): p = 2^(s*scale*log2e - m).  The reference max m of a row is the one of the EARLIER
// key blocks, so no max -> exp dependency sits on the critical path; how far the current block
// outgrew it is read off the block's row sum afterwards (max p <= sum p):
//   sum <= 2^8      : nothing to do (lazy rescale; the final O/l uses the same m, so this is exact)
//   sum <  2^100    : this block's P and row sum stay relative to the old m (exact); before the next
//                     block m is raised by D = floor(log2 sum) + 1 and O_t (TMEM), l are multiplied by 2^-D
//   otherwise       : (exponentials may have overflowed) the item is flagged and redone by the
//                     kSafe instantiation of this kernel, which takes the exact row max before the
//                     exponentials of every block; it is launched right after and returns at once
//                     when nothing was flagged.
// The first key block of an item always takes the exact-max path.
//
// TMEM (512 columns): S_0 [0,128)  S_1 [128,256)  O_0 [256,384)  O_1 [384,512); P_t (bf16) aliases
// columns [0,32) and [64,96) of S_t (tensor-pipe ops run in issue order, so S_t(next) is issued after
// O_t += P_t V(prev) and may overwrite it).
//
// Key blocks of an item: first the merged TOPK union of the pair (per entry a 2-bit mask says which
// tile attends it), then SINK, then CUR (both tiles).  All K/V come from the ctx cache.  In paper-mask
// mode (uf_select_blocks_paper) there is no SINK and no implicit CUR: every kept block, the query
// block's own included, is in the lists, with its valid-row count.
#include "uf_internal.h"
#include "uf_sm100_ptx.h"

namespace {

constexpr int kNK = 3;                 // K ring stages
constexpr int kNV = 2;                 // V ring stages
constexpr int kTile = 128 * 128 * 2;   // bytes of one 128 x 128 bf16 tile
constexpr int kHalf = kTile / 2;       // one 64-column box
constexpr int kThreads = 384;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: below this growth of the row max, keep m
constexpr float kPanicSum = 1.2676506e30f;   // 2^100: a block row sum at or above this -> redo the item in the safe kernel
constexpr uint32_t kPArrivals = 8;          // one lane of each of the 8 softmax warps arrives on P_FULL

// smem carve-up (offsets from a 1024-aligned base)
constexpr int kOffQ = 0;                          // 2 tiles
constexpr int kOffK = kOffQ + 2 * kTile;
constexpr int kOffV = kOffK + kNK * kTile;
constexpr int kOffBar = kOffV + kNV * kTile;
constexpr int kNumBars = 4 + 2 * kNK + 2 * kNV + 6;
constexpr int kOffTmemPtr = kOffBar + kNumBars * 8;
constexpr int kOffXc = kOffTmemPtr + 16;              // softmax row-pair exchange: [tile][half][row][parity] bytes
constexpr int kSmemBytes = kOffXc + 2 * 2 * 128 * 2 + 1024;   // + alignment slack
static_assert(kSmemBytes <= 232448, "more than 227 KB of shared memory");

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
// Shared-memory matrix descriptors, 128-byte swizzle.  The upper 32 bits are the same for every operand
// here (SBO = 1024 B between 8-row groups, version 1, swizzle mode 2); the lower 32 bits are
// (address >> 4) | (LBO >> 4) << 16, i.e. a per-buffer base plus a small constant per K step.
constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
__device__ __forceinline__ uint32_t desc_lo(uint32_t saddr, uint32_t lbo_bytes) {
  return ((saddr & 0x3FFFFu) >> 4) | ((lbo_bytes >> 4) << 16);
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      ".reg .b64 da, db;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "mov.b64 da, {%1, %5};\n\t"
      "mov.b64 db, {%2, %5};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %3, p;\n\t"
      "}" ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(idesc), "r"(acc), "r"(kDescHi) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      ".reg .b64 db;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "mov.b64 db, {%2, %5};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %3, p;\n\t"
      "}" ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(idesc), "r"(acc), "r"(kDescHi) : "memory");
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

#define UF_TMEM_ST16(taddr, a)                                                                                 \
  asm volatile(                                                                                                \
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "                                                          \
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"                               \
      ::"r"(taddr), "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]), "r"(a[7]),    \
        "r"(a[8]), "r"(a[9]), "r"(a[10]), "r"(a[11]), "r"(a[12]), "r"(a[13]), "r"(a[14]), "r"(a[15])           \
      : "memory")

// tcgen05.wait::ld that also names the 32 destination registers of the load it completes, so that no use
// of them can be scheduled above it (the load itself returns before its registers are written).
#define UF_TMEM_WAIT_LD32(a)                                                                                   \
  asm volatile("tcgen05.wait::ld.sync.aligned;"                                                                \
      : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]),        \
        "+r"(a[8]), "+r"(a[9]), "+r"(a[10]), "+r"(a[11]), "+r"(a[12]), "+r"(a[13]), "+r"(a[14]), "+r"(a[15]),  \
        "+r"(a[16]), "+r"(a[17]), "+r"(a[18]), "+r"(a[19]), "+r"(a[20]), "+r"(a[21]), "+r"(a[22]),             \
        "+r"(a[23]), "+r"(a[24]), "+r"(a[25]), "+r"(a[26]), "+r"(a[27]), "+r"(a[28]), "+r"(a[29]),             \
        "+r"(a[30]), "+r"(a[31])                                                                               \
      :: "memory")

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

__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
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
// x is clamped to [-126, 126] by ONE instruction (min.xorsign.abs -> FMNMX.XORSIGN): below, because the
// polynomial can return 1 - 7.5e-5 (exponent field 126, so floor(x) = -127 would wrap); above, because for
// x >= 129 the exponent add would wrap into the sign bit and silently return a small or negative number.
// A clamped 2^126 makes the row sum >= 2^100, so the item takes the panic path (redo with the exact max).
constexpr int kEmuPairs = 3;
__device__ __forceinline__ constexpr bool pair_emulated(int j) { return ((j & 7) * kEmuPairs) % 8 < kEmuPairs; }

__device__ __forceinline__ float clamp126(float x) {       // sign(x) * min(|x|, 126)
  float y;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(y) : "f"(x), "f"(126.0f));
  return y;
}
__device__ __forceinline__ uint64_t ex2_pair(uint64_t x, bool emulate) {
  float x0, x1;
  unpack2(x, x0, x1);
  if (!emulate) return pack2(ex2(x0), ex2(x1));
  const uint64_t magic = pack2(12582912.0f, 12582912.0f);            // 2^23 + 2^22
  x = pack2(clamp126(x0), clamp126(x1));
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

// One 32-column chunk of a softmax pass: p = 2^(s*sl2 - m) as bf16 pairs into pk[] and fp32 row sums into
// the two packed accumulators.  The row sum adds the bf16-ROUNDED probabilities, the very numbers the P V MMA
// multiplies, so O = sum(P~ v) / sum(P~) is a consistent weighted mean whatever the rounding of P~ (a one-hot
// row returns its V row exactly; with the unrounded sum it carried the 2^-8 relative rounding error of its
// single probability, which is not 1 under a stale reference max).  `chunk` (0..3, position in the 128-key block) selects which column pairs
// take the polynomial (unused: the pattern has period 8 pairs); `nvalid_left` < 32 masks the tail of a ragged key block (R-3).
__device__ __forceinline__ void exp_chunk(uint32_t (&s)[32], uint32_t (&pk)[16], int chunk, int nvalid_left,
                                          uint64_t sl22, uint64_t nm2, uint64_t& acc0, uint64_t& acc1) {
  if (nvalid_left < 32) {
#pragma unroll
    for (int c = 0; c < 32; ++c)
      if (c >= nvalid_left) s[c] = 0xff800000u;          // -inf
  }
#pragma unroll
  for (int u = 0; u < 32; u += 2) {
    const int j = (u >> 1);                               // pattern repeats every 8 pairs
    const uint64_t x = fma2(pack2(__uint_as_float(s[u]), __uint_as_float(s[u + 1])), sl22, nm2);
    const uint64_t p = ex2_pair(x, pair_emulated(j));
    float p0, p1;
    unpack2(p, p0, p1);
    const uint32_t w = pack_bf16x2(p0, p1);
    pk[u >> 1] = w;
    // add.rn.f32.bf16 (FHADD.BF16 with a half-register select): fp32 accumulator += one bf16 half of w, one
    // instruction per element and no unpacking (measured against widening with shift / mask + packed add)
    {
      float a0, a1;
      uint64_t& acc = (j & 1) ? acc1 : acc0;
      unpack2(acc, a0, a1);
      unsigned short lo, hi;
      asm("mov.b32 {%0, %1}, %2;" : "=h"(lo), "=h"(hi) : "r"(w));
      asm("add.rn.f32.bf16 %0, %1, %0;" : "+f"(a0) : "h"(lo));
      asm("add.rn.f32.bf16 %0, %1, %0;" : "+f"(a1) : "h"(hi));
      acc = pack2(a0, a1);
    }
  }
}

// upper 16 bits of x rounded toward +infinity (a bf16 >= x); -inf stays -inf
__device__ __forceinline__ uint32_t bf16_bits_up(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u >> 16) + (((u & 0xffffu) != 0u && x > 0.f) ? 1u : 0u);
}

// instruction descriptor kind::f16: D fp32, A/B bf16, M = N = 128; B MN-major for P V
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescQK | (1u << 16);

struct AttnParams {
  const int32_t* sel_pair;   // [H][NP][2*kcap]
  const int32_t* pair_cnt;   // [H][NP]
  float* lse;                // [H][ntok] or null
  int32_t* panic_item;       // [H * np_cur]: == seq when the item must be redone by the safe kernel
  int32_t* panic_last;       // == seq when any item of this launch was flagged
  int32_t seq;               // launch sequence number (never 0)
  int H, NP, kcap, np_cur;
  int ntok, nqb;
  int n_sink, sink_ntok;
  int n_cur;                 // CUR blocks every query block attends implicitly (nqb; 0 in paper-mask mode: all in the lists)
  int cur_phys0;
  float sl2;                 // softmax scale * log2(e)
};

template <bool kSafe>
__global__ void __launch_bounds__(kThreads, 1)
uf_attn_sm100_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_o,
                     const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                     const AttnParams a) {
  if (kSafe && *a.panic_last != a.seq) return;         // nothing was flagged: the usual case
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

  // An item = (head h, query-block pair p).  Its key blocks: the pair's merged TOPK list (n_u entries,
  // loaded 32 at a time, one per lane, and broadcast by shuffle), then n_sink SINK blocks, then nqb CUR
  // blocks.  The safe kernel only takes the items the fast kernel flagged.
#define UF_ITEM_LOOP_BEGIN                                                                      \
  for (int it = blockIdx.x; it < n_items; it += gridDim.x) {                                    \
    if (kSafe && a.panic_item[it] != a.seq) continue;                                           \
    const int h = it / a.np_cur, p = it % a.np_cur;                                             \
    const int64_t pi = (int64_t)h * a.NP + p;                                                   \
    const int n_u = __shfl_sync(0xffffffffu, a.pair_cnt[pi], 0);                                \
    const int32_t* ulist = a.sel_pair + pi * 2 * a.kcap;                                        \
    const int full_mask = (2 * p + 1 < a.nqb) ? 3 : 1;
#define UF_ITEM_LOOP_END }

  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
    if (warp == 8) {
      // ================================ TMA producer ================================
      uint32_t ks = 0, kph = 0, vs = 0, vph = 0, qph0 = 0, qph1 = 0;
      auto load_kv = [&](int phys, int h) {
        const int row = phys * 128;
        {
          const uint32_t bf = bars + (K_FULL0 + ks) * 8, dst = base + kOffK + ks * kTile;
          mbar_wait(bars + (K_EMPTY0 + ks) * 8, kph ^ 1);
          if (elect_one()) {
            mbar_expect_tx(bf, kTile);
            tma_load_3d(dst, &tm_k, bf, 0, row, h);
            tma_load_3d(dst + kHalf, &tm_k, bf, 64, row, h);
          }
          if (++ks == kNK) { ks = 0; kph ^= 1; }
        }
        {
          const uint32_t bf = bars + (V_FULL0 + vs) * 8, dst = base + kOffV + vs * kTile;
          mbar_wait(bars + (V_EMPTY0 + vs) * 8, vph ^ 1);
          if (elect_one()) {
            mbar_expect_tx(bf, kTile);
            tma_load_3d(dst, &tm_v, bf, 0, row, h);
            tma_load_3d(dst + kHalf, &tm_v, bf, 64, row, h);
          }
          if (++vs == kNV) { vs = 0; vph ^= 1; }
        }
      };
      UF_ITEM_LOOP_BEGIN
        int32_t nxt = (lane < n_u) ? __ldg(ulist + lane) : 0;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (!(full_mask & (1 << t))) continue;
          const uint32_t bq = bars + (Q_FULL0 + t) * 8;
          uint32_t& qph = t ? qph1 : qph0;
          mbar_wait(bars + (Q_EMPTY0 + t) * 8, qph ^ 1);
          qph ^= 1;
          const int row0 = (2 * p + t) * 128;
          if (elect_one()) {
            mbar_expect_tx(bq, kTile);
            tma_load_3d(base + kOffQ + t * kTile, &tm_q, bq, 0, row0, h);
            tma_load_3d(base + kOffQ + t * kTile + kHalf, &tm_q, bq, 64, row0, h);
          }
        }
        for (int st0 = 0; st0 < n_u; st0 += 32) {
          const int32_t mine = nxt;
          if (st0 + 32 + lane < n_u) nxt = __ldg(ulist + st0 + 32 + lane);
          const int cnt = min(32, n_u - st0);
          for (int j = 0; j < cnt; ++j) load_kv(uf_entry_phys(__shfl_sync(0xffffffffu, mine, j)), h);
        }
        for (int j = 0; j < a.n_sink; ++j) load_kv(j, h);
        for (int j = 0; j < a.n_cur; ++j) load_kv(a.cur_phys0 + j, h);
      UF_ITEM_LOOP_END
    } else if (warp == 9) {
      // ================================ MMA issuer ==================================
      // Per key block and attending tile t: O_t += P_t V of the PREVIOUS block of that tile (once its
      // P is ready), then S_t = Q_t K^T of this block.  Tensor-pipe order per step with both tiles:
      // PV_0(n-1) QK_0(n) PV_1(n-1) QK_1(n): while the softmax warps of one tile work, the pipe runs
      // the other tile.
      const uint32_t q_lo0 = desc_lo(base + kOffQ, 16), q_lo1 = desc_lo(base + kOffQ + kTile, 16);
      const uint32_t k_lo_base = desc_lo(base + kOffK, 16);
      const uint32_t v_lo_base = desc_lo(base + kOffV, kHalf);
      static_assert(kNV == 2, "vrem0/vrem1 below assume a 2-stage V ring");
      uint32_t ks = 0, kph = 0, vs = 0, vph = 0, qph0 = 0, qph1 = 0, pph0 = 0, pph1 = 0;
      int vrem0 = 0, vrem1 = 0;                      // tiles that still have to consume V stage 0 / 1
      bool pend[2] = {false, false}, first_pv[2] = {true, true};
      uint32_t pend_vs[2] = {0, 0}, pend_vph[2] = {0, 0};

      auto do_pv = [&](int t) {
        uint32_t& pph = t ? pph1 : pph0;
        mbar_wait(bars + (P_FULL0 + t) * 8, pph);
        pph ^= 1;
        const uint32_t pvs = pend_vs[t];
        mbar_wait(bars + (V_FULL0 + pvs) * 8, pend_vph[t]);
        tc_fence_after();
        const int left = (pvs == 0) ? --vrem0 : --vrem1;
        if (elect_one()) {
          // B = V tile, MN-major: 8-key groups 1024 B apart (SBO), the two 64-column halves 16 KB apart (LBO)
          const uint32_t v_lo = v_lo_base + pvs * (kTile >> 4);
          const uint32_t d_tmem = tmem + 256 + t * 128, p_tmem = tmem + t * 128;
#pragma unroll
          for (int k = 0; k < 8; ++k)
            // keys [16k, 16k + 16) of P_t: the thread pair's halves sit at S_t columns [0, 32) and [64, 96)
            mma_ts(d_tmem, p_tmem + (k >> 2) * 64 + (k & 3) * 8, v_lo + k * (2048 >> 4), kIdescPV,
                   (first_pv[t] && k == 0) ? 0u : 1u);
          if (left == 0) tc_commit(bars + (V_EMPTY0 + pvs) * 8);
        }
        first_pv[t] = false;
        pend[t] = false;
      };

      auto step = [&](int m) {
        mbar_wait(bars + (K_FULL0 + ks) * 8, kph);
        tc_fence_after();
        const uint32_t k_lo = k_lo_base + ks * (kTile >> 4);
        int users = 0;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (!(m & (1 << t))) continue;
          if (pend[t]) do_pv(t);
          if (elect_one()) {
            const uint32_t q_lo = t ? q_lo1 : q_lo0;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              // K-major operands: 8-row groups 1024 B apart (SBO); 16 elements = 32 B along K, second half +16 KB
              const uint32_t koff = ((k & 3) * 32 + (k >> 2) * kHalf) >> 4;
              mma_ss(tmem + t * 128, q_lo + koff, k_lo + koff, kIdescQK, k == 0 ? 0u : 1u);
            }
            tc_commit(bars + (S_FULL0 + t) * 8);
          }
          pend[t] = true; pend_vs[t] = vs; pend_vph[t] = vph;
          ++users;
        }
        if (elect_one()) tc_commit(bars + (K_EMPTY0 + ks) * 8);
        if (vs == 0) vrem0 = users; else vrem1 = users;
        if (++ks == kNK) { ks = 0; kph ^= 1; }
        if (++vs == kNV) { vs = 0; vph ^= 1; }
#pragma unroll
        for (int t = 0; t < 2; ++t)
          if (!(m & (1 << t)) && pend[t]) do_pv(t);      // keep V stages flowing (no deadlock)
      };

      UF_ITEM_LOOP_BEGIN
        int32_t nxt = (lane < n_u) ? __ldg(ulist + lane) : 0;
        first_pv[0] = first_pv[1] = true;
        if (full_mask & 1) { mbar_wait(bars + Q_FULL0 * 8, qph0); qph0 ^= 1; }
        if (full_mask & 2) { mbar_wait(bars + Q_FULL1 * 8, qph1); qph1 ^= 1; }
        for (int st0 = 0; st0 < n_u; st0 += 32) {
          const int32_t mine = nxt;
          if (st0 + 32 + lane < n_u) nxt = __ldg(ulist + st0 + 32 + lane);
          const int cnt = min(32, n_u - st0);
          for (int j = 0; j < cnt; ++j) step(uf_entry_mask(__shfl_sync(0xffffffffu, mine, j)));
        }
        for (int j = 0; j < a.n_sink + a.n_cur; ++j) step(full_mask);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (pend[t]) do_pv(t);
          if ((full_mask & (1 << t)) && elect_one()) tc_commit(bars + (O_FULL0 + t) * 8);
        }
      UF_ITEM_LOOP_END
    }
  } else {
    // ================================== softmax + epilogue ==================================
    // All 8 warps work on ONE tile at a time (tile 0 and tile 1 alternate, in the order the MMA warp
    // produces S_0 / S_1): a query row is shared by two threads, lane `lane` of warps wq and wq + 4
    // (both may touch TMEM lanes [32 wq, 32 wq + 32)); the thread with half = 0 owns S columns (keys)
    // [0, 64) and O columns [0, 64), the other one [64, 128).  So every scheduler always has two warps
    // on the same softmax step and the step takes half as long as with one thread per row.
    // The two threads of a row must use the same reference max m: after a step each publishes in shared
    // memory by how many binades D its partial row sum exceeds 2^8 (one byte, 0 = not at all; slots
    // double-buffered by step parity because the partner may be one step ahead); both read the other's
    // before their next step of that tile (the P_FULL -> S_FULL chain orders the accesses) and raise m by
    // the larger D: the same number on both sides, and O_t, l are rescaled by an exact power of two.
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    const int wq = warp & 3;                           // TMEM lane quarter
    const int half = warp >> 2;                        // which 64 keys of a block / 64 columns of O
    const int row = wq * 32 + lane;                    // row in the tile == TMEM lane
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    const uint32_t col0 = (uint32_t)half * 64;
    const float sl2 = a.sl2;
    const uint64_t sl22 = pack2(sl2, sl2);
    volatile uint8_t* xc = reinterpret_cast<volatile uint8_t*>(base_ptr + kOffXc);     // [tile][half][row][parity]
    uint32_t sph0 = 0, sph1 = 0, oph0 = 0, oph1 = 0;

    UF_ITEM_LOOP_BEGIN
      // per tile: reference max, partial row sum (this thread's keys), own published D, step parity
      float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
      int d0 = 0, d1 = 0, par0 = 0, par1 = 0;
      bool first0 = true, first1 = true;

      auto softmax_step = [&](const int t, float& m, float& l, int& d_own, int& par, bool& first, uint32_t& sph,
                              int nvalid) {
        const uint32_t s_tmem = tmem + lane_addr + t * 128 + col0;          // this thread's 64 S columns
        const uint32_t o_tmem = tmem + lane_addr + 256 + t * 128 + col0;    // and its 64 O columns
        volatile uint8_t* x_own = xc + ((t * 2 + half) * 128 + row) * 2;
        volatile uint8_t* x_oth = xc + ((t * 2 + (half ^ 1)) * 128 + row) * 2;
        const int left = nvalid - (int)col0;                                // valid keys in this thread's half
        // multiply this thread's half of the O_t row by f (O_t is quiescent between S_FULL and our
        // P_FULL arrive: the commit behind S_FULL also covers the earlier O_t += P_t V)
        auto rescale_o = [&](float f) {
#pragma unroll
          for (int cc = 0; cc < 64; cc += 32) {
            uint32_t ov[32];
            UF_TMEM_LD32(o_tmem + cc, ov, 0);
            UF_TMEM_WAIT_LD32(ov);
#pragma unroll
            for (int c = 0; c < 32; ++c) ov[c] = __float_as_uint(__uint_as_float(ov[c]) * f);
            UF_TMEM_ST32(o_tmem + cc, ov, 0);
          }
        };
        mbar_wait(bars + (S_FULL0 + t) * 8, sph);
        sph ^= 1;
        tc_fence_after();
        uint32_t sa[32], sb[32], pk[16];
        const bool exact = kSafe || first;
        if (!kSafe && !first) {
          // deferred raise of m by D binades: the larger of what the two threads of the row published
          // after the previous step of this tile
          const int D = max(d_own, (int)x_oth[par ^ 1]);
          if (__any_sync(0xffffffffu, D > 0)) {
            const float f = __int_as_float((127 - D) << 23);                // 2^-D (D <= 101), 1 if D == 0
            rescale_o(f);
            l *= f;
            m += (float)D;
          }
        }
        if (exact) {
          // exact row max BEFORE the exponentials: first key block of an item / every block when kSafe.
          // The halves are exchanged as bf16 (both threads then hold the same number).
          float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            UF_TMEM_LD32(s_tmem + c * 32, sa, 0);
            UF_TMEM_WAIT_LD32(sa);
#pragma unroll
            for (int u = 0; u < 32; u += 2) {
              const float v0 = (c * 32 + u < left) ? __uint_as_float(sa[u]) : -INFINITY;
              const float v1 = (c * 32 + u + 1 < left) ? __uint_as_float(sa[u + 1]) : -INFINITY;
              if (u & 2) mx1 = max3(mx1, v0, v1); else mx0 = max3(mx0, v0, v1);
            }
          }
          const uint32_t mine = bf16_bits_up(fmaxf(mx0, mx1));
          *reinterpret_cast<volatile uint16_t*>(x_own) = (uint16_t)mine;
          asm volatile("bar.sync %0, 64;" ::"r"(2 + wq) : "memory");
          const uint32_t theirs = *reinterpret_cast<volatile uint16_t*>(x_oth);
          const float rowmax = fmaxf(__uint_as_float(mine << 16), __uint_as_float(theirs << 16));
          asm volatile("bar.sync %0, 64;" ::"r"(2 + wq) : "memory");     // both have read: the slot may be reused
          const float m_new = fmaxf(m, rowmax * sl2);
          if (first) {
            m = m_new;
            first = false;
          } else {
            const bool need = (m_new - m) > kRescaleThreshold;
            if (__any_sync(0xffffffffu, need)) {
              const float f = need ? ex2(m - m_new) : 1.0f;
              if (need) { m = m_new; l *= f; }
              rescale_o(f);
            }
          }
        }
        // exponentials of this thread's 64 keys: chunk 1 in flight while chunk 0 is processed; the P chunks
        // go to columns [col0, col0 + 32) of S_t, which are in registers by then
        const uint64_t nm2 = pack2(-m, -m);
        uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
        UF_TMEM_LD32(s_tmem + 0, sa, 0);
        UF_TMEM_WAIT_LD32(sa);
        UF_TMEM_LD32(s_tmem + 32, sb, 0);
        exp_chunk(sa, pk, half * 2 + 0, left, sl22, nm2, acc0, acc1);
        UF_TMEM_ST16(s_tmem + 0, pk);
        UF_TMEM_WAIT_LD32(sb);
        exp_chunk(sb, pk, half * 2 + 1, left - 32, sl22, nm2, acc0, acc1);
        UF_TMEM_ST16(s_tmem + 16, pk);
        float a0, a1, b0, b1;
        unpack2(acc0, a0, a1);
        unpack2(acc1, b0, b1);
        const float lsum = (a0 + a1) + (b0 + b1);
        l += lsum;
        if (!kSafe) {
          // p <= lsum, so while the partial row sum stays below 2^8 no exponent exceeded 8 and m can stay;
          // otherwise propose to raise m by D = floor(log2 lsum) + 1 binades (m + D > the true max of these keys).
          int D = 0;
          if (!(lsum <= 256.0f)) {
            if (lsum < kPanicSum) {
              D = (int)((__float_as_uint(lsum) >> 23) & 0xffu) - 126;      // floor(log2 lsum) + 1
            } else {                                    // (also inf / NaN) exponentials may have overflowed
              a.panic_item[it] = a.seq;
              *a.panic_last = a.seq;
              D = 101;
            }
          }
          x_own[par] = (uint8_t)D;
          d_own = D;
        }
        par ^= 1;
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bars + (P_FULL0 + t) * 8);
      };

      // ---- the item's key blocks, in the MMA warp's order: per block tile 0 then tile 1 ----
      {
        int32_t mine = 0;
        for (int st = 0; st < n_u; ++st) {
          if ((st & 31) == 0) mine = (st + lane < n_u) ? __ldg(ulist + st + lane) : 0;
          const int32_t e = __shfl_sync(0xffffffffu, mine, st & 31);
          const int msk = uf_entry_mask(e), nvalid = uf_entry_nvalid(e);
          if (msk & 1) softmax_step(0, m0, l0, d0, par0, first0, sph0, nvalid);
          if (msk & 2) softmax_step(1, m1, l1, d1, par1, first1, sph1, nvalid);
        }
        for (int j = 0; j < a.n_sink + a.n_cur; ++j) {
          const int nvalid = (j < a.n_sink) ? min(128, a.sink_ntok - j * 128) : min(128, a.ntok - (j - a.n_sink) * 128);
          softmax_step(0, m0, l0, d0, par0, first0, sph0, nvalid);
          if (full_mask & 2) softmax_step(1, m1, l1, d1, par1, first1, sph1, nvalid);
        }
      }

      // ---- epilogue per tile: O_t / l -> bf16 -> swizzled staging (the Q_t buffer) -> TMA store ----
      // (a raise of m still pending here is dropped: O_t / l does not depend on it, and m, l stay consistent)
      auto epilogue = [&](const int t, float m, float l, uint32_t& oph) {
        const uint32_t o_tmem = tmem + lane_addr + 256 + t * 128 + col0;
        unsigned char* stage = base_ptr + kOffQ + t * kTile;
        mbar_wait(bars + (O_FULL0 + t) * 8, oph);      // every MMA of the item is complete: Q_t is free too
        oph ^= 1;
        tc_fence_after();
        // total row sum = the two threads' partial sums (exchanged through the staging buffer)
        volatile float* xl = reinterpret_cast<volatile float*>(stage);
        xl[half * 128 + row] = l;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const float l_tot = l + xl[(half ^ 1) * 128 + row];
        asm volatile("bar.sync 1, 256;" ::: "memory");                     // all read before the staging writes
        const float inv = 1.0f / l_tot;
#pragma unroll
        for (int cc = 0; cc < 64; cc += 32) {
          uint32_t ov[32];
          UF_TMEM_LD32(o_tmem + cc, ov, 0);
          UF_TMEM_WAIT_LD32(ov);
          unsigned char* half_base = stage + half * kHalf + row * 128;     // 64-column box `half` of the tile
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 w;
            w.x = pack_bf16x2(__uint_as_float(ov[8 * j + 0]) * inv, __uint_as_float(ov[8 * j + 1]) * inv);
            w.y = pack_bf16x2(__uint_as_float(ov[8 * j + 2]) * inv, __uint_as_float(ov[8 * j + 3]) * inv);
            w.z = pack_bf16x2(__uint_as_float(ov[8 * j + 4]) * inv, __uint_as_float(ov[8 * j + 5]) * inv);
            w.w = pack_bf16x2(__uint_as_float(ov[8 * j + 6]) * inv, __uint_as_float(ov[8 * j + 7]) * inv);
            const int chunk = (cc >> 3) + j;                               // 16-byte chunk within the 128-byte row
            *reinterpret_cast<uint4*>(half_base + ((chunk ^ (row & 7)) << 4)) = w;
          }
        }
        tc_fence_before();
        fence_proxy_async();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const int row0 = (2 * p + t) * 128;
        if (warp == 0 && lane == 0) {
          const uint32_t src = base + kOffQ + t * kTile;
          tma_store_3d(&tm_o, src, 0, row0, h);
          tma_store_3d(&tm_o, src + kHalf, 64, row0, h);
          tma_store_commit_and_wait_read();
          mbar_arrive(bars + (Q_EMPTY0 + t) * 8);
        }
        if (half == 0 && a.lse != nullptr && row0 + row < a.ntok)
          a.lse[(int64_t)h * a.ntok + row0 + row] = (m + log2f(l_tot)) * 0.6931471805599453f;
      };
      epilogue(0, m0, l0, oph0);
      if (full_mask & 2) epilogue(1, m1, l1, oph1);
    UF_ITEM_LOOP_END
    if (warp == 0 && lane == 0) tma_store_wait_all();
  }
#undef UF_ITEM_LOOP_BEGIN
#undef UF_ITEM_LOOP_END

  tc_fence_before();
  __syncthreads();
  if (warp == 10) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

// =====================================================================================================
// CTA-pair variant (cta_group::2): ONE 128-row query tile per CTA, the two CTAs of a cluster take query blocks
// (2p, 2p+1) of an item and act as one 256-row MMA tile.
//   * every K tile is split between the pair by key (CTA r holds keys [64 r, 64 r + 64)), every V tile by column
//     (CTA r holds columns [64 r, 64 r + 64) of all 128 keys): each SM ingests 32 KB per key block for its tile, as
//     the two-tiles-per-CTA kernel does, and reads half as much operand data from shared memory per MMA;
//   * S is TRIPLE-BUFFERED in TMEM (S_0 [0,128), S_1 [128,256), S_2 [256,384), O [384,512)): S(n+3) = Q K(n+3)^T is
//     issued right after O += P(n) V(n), so softmax(n+1) and softmax(n+2) find their S ready and the tensor pipe
//     never waits for the softmax of the block it just fed: no softmax -> PV -> QK chain any more.  P(n) aliases
//     S(n mod 3).  (Two buffers were measured first: the loop P_FULL(n) -> PV(n), QK(n+2) -> S_FULL(n+2) carries the
//     cross-CTA barrier latencies, about 1000 cycles per turn, and two steps of slack do not cover it: 1610 cycles
//     per block; three do.)
//   * both CTAs walk the pair's merged list; a block only the other tile attends is a zero-fill step (P = 0).
//   * a raise of the reference max decided after block n is applied at the START of step n+1 to m and l, and to O at
//     the END of step n+1 (O += P(n) V is still in flight at its start; P(n+1) is already relative to the new m and
//     O += P(n+1) V is issued only after this step's P_FULL arrive).
// Barriers: TMA loads of both CTAs complete on the LEADER's Q/K/V_FULL; tcgen05.commit multicasts S_FULL, PV_DONE,
// O_FULL and the ring's EMPTY barriers to both CTAs; the softmax warps of both CTAs arrive on the leader's P_FULL.
constexpr int kNK2 = 6;                  // K ring stages (half tiles)
constexpr int kNV2 = 4;                  // V ring stages (half tiles)
constexpr int kHalfTile = kTile / 2;     // this CTA's half of a K or V tile
constexpr int kOff2Q = 0;
constexpr int kOff2K = kOff2Q + kTile;
constexpr int kOff2V = kOff2K + kNK2 * kHalfTile;
constexpr int kOff2Bar = kOff2V + kNV2 * kHalfTile;
enum Bar2 {
  B2_Q_FULL = 0, B2_Q_EMPTY,
  B2_K_FULL0 = 2, B2_K_EMPTY0 = B2_K_FULL0 + kNK2,
  B2_V_FULL0 = B2_K_EMPTY0 + kNK2, B2_V_EMPTY0 = B2_V_FULL0 + kNV2,
  B2_S_FULL0 = B2_V_EMPTY0 + kNV2, B2_P_FULL0 = B2_S_FULL0 + 3, B2_PV_DONE0 = B2_P_FULL0 + 3, B2_O_FULL = B2_PV_DONE0 + 2,
  B2_DEC0, kNumBars2 = B2_DEC0 + 2           // DEC[gs & 1]: step gs of a two-group kernel has published its decision
};
constexpr int kOff2TmemPtr = kOff2Bar + kNumBars2 * 8;
constexpr int kOff2Xc = kOff2TmemPtr + 16;                    // row-pair exchange: [group][half][row][parity] bytes
constexpr int kOff2M0 = kOff2Xc + 2 * 2 * 128 * 2;            // two softmax groups: reference max of the item's rows (float)
constexpr int kOff2Rc = kOff2M0 + 128 * 4;                    // ... binades it was raised by so far (int)
constexpr int kOff2Cnt = kOff2Rc + 128 * 4;                   // ... steps whose start decision is published
constexpr int kSmemBytes2 = kOff2Cnt + 16 + 1024;
constexpr uint32_t kIdescQK2 = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((256u >> 4) << 24);
constexpr uint32_t kIdescPV2 = kIdescQK2 | (1u << 16);

// kGroups = 2 (fast kernel only): TWO groups of 8 softmax warps take the key blocks of the tile in turn (group g the
// blocks with global step number gs = g mod 2), so that the TMEM round trips, barrier waits and dependency stalls of
// one group's step run under the arithmetic of the other's (the arithmetic alone needs ~1000-1080 cycles per block
// and 8 warps cannot overlap the ~320 cycles around it).  Both groups use ONE reference max per row, m = m0 + r
// (m0 set by the group that gets the first attended block, r = binades raised so far, both in shared memory): a step
// publishes its decision (a raise of r) before it computes, and the next step, the other group's, starts only after
// that, so every P is relative to the m that O will have when its O += P V is issued.
template <bool kSafe, int kGroups>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__((8 * kGroups + 4) * 32, 1)
uf_attn_pair_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_o,
                    const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                    const AttnParams a) {
  if (kSafe && *a.panic_last != a.seq) return;         // nothing was flagged (both CTAs of a pair see the same value)
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + kOff2Bar;
  volatile uint32_t* tmem_ptr_smem = reinterpret_cast<volatile uint32_t*>(base_ptr + kOff2TmemPtr);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)ufptx::cluster_ctarank();      // 0 = leader: issues every MMA of the pair
  const int pair = (int)(blockIdx.x >> 1), n_pairs = (int)(gridDim.x >> 1);
  const int n_items = a.H * a.np_cur;
  static_assert(kGroups == 1 || !kSafe, "the exact-max kernel runs one softmax group");
  constexpr int kW0 = 8 * kGroups;                     // first non-softmax warp: producer, MMA issuer, TMEM allocator
  if (threadIdx.x == 0) *reinterpret_cast<volatile uint32_t*>(base_ptr + kOff2Cnt) = 0u;

  if (warp == kW0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_o));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_k));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_v));
  }
  if (warp == kW0 + 1 && lane == 0) {
    for (int i = 0; i < kNumBars2; ++i)
      mbar_init(bars + i * 8, (i >= B2_P_FULL0 && i < B2_P_FULL0 + 3) ? 2 * kPArrivals : 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  if (warp == kW0 + 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32((const void*)tmem_ptr_smem)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  ufptx::cluster_sync();                               // the peer's barriers exist before anything signals them
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_smem;

#define UF_ITEM_LOOP_BEGIN                                                                      \
  for (int it = pair; it < n_items; it += n_pairs) {                                            \
    if (kSafe && a.panic_item[it] != a.seq) continue;                                           \
    const int h = it / a.np_cur, p = it % a.np_cur;                                             \
    const int64_t pi = (int64_t)h * a.NP + p;                                                   \
    const int n_u = __shfl_sync(0xffffffffu, a.pair_cnt[pi], 0);                                \
    const int32_t* ulist = a.sel_pair + pi * 2 * a.kcap;                                        \
    const int full_mask = (2 * p + 1 < a.nqb) ? 3 : 1;
#define UF_ITEM_LOOP_END }

  if (warp >= kW0) {
    if (kGroups == 1) asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == kW0) {
      // ================================ TMA producer (both CTAs) =====================
      uint32_t ks = 0, kph = 0, vs = 0, vph = 0, qph = 0;
      auto load_kv = [&](int phys, int h) {
        {
          const uint32_t bf = bars + (B2_K_FULL0 + ks) * 8, dst = base + kOff2K + ks * kHalfTile;
          mbar_wait(bars + (B2_K_EMPTY0 + ks) * 8, kph ^ 1);
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(bf, 2 * kHalfTile);            // both CTAs' halves land on the leader's barrier
            const int row = phys * 128 + rank * 64;                     // this CTA's 64 keys
            ufptx::tma_load_3d_2sm(dst, &tm_k, bf, 0, row, h);
            ufptx::tma_load_3d_2sm(dst + kHalfTile / 2, &tm_k, bf, 64, row, h);
          }
          if (++ks == kNK2) { ks = 0; kph ^= 1; }
        }
        {
          const uint32_t bf = bars + (B2_V_FULL0 + vs) * 8, dst = base + kOff2V + vs * kHalfTile;
          mbar_wait(bars + (B2_V_EMPTY0 + vs) * 8, vph ^ 1);
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(bf, 2 * kHalfTile);
            ufptx::tma_load_3d_2sm(dst, &tm_v, bf, rank * 64, phys * 128, h);   // this CTA's 64 columns of all 128 keys
          }
          if (++vs == kNV2) { vs = 0; vph ^= 1; }
        }
      };
      UF_ITEM_LOOP_BEGIN
        (void)full_mask;
        int32_t nxt = (lane < n_u) ? __ldg(ulist + lane) : 0;
        {
          const uint32_t bq = bars + B2_Q_FULL * 8;
          mbar_wait(bars + B2_Q_EMPTY * 8, qph ^ 1);
          qph ^= 1;
          const int row0 = (2 * p + rank) * 128;                        // past the last token (no such tile): zero-filled
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(bq, 2 * kTile);
            ufptx::tma_load_3d_2sm(base + kOff2Q, &tm_q, bq, 0, row0, h);
            ufptx::tma_load_3d_2sm(base + kOff2Q + kHalf, &tm_q, bq, 64, row0, h);
          }
        }
        for (int st0 = 0; st0 < n_u; st0 += 32) {
          const int32_t mine = nxt;
          if (st0 + 32 + lane < n_u) nxt = __ldg(ulist + st0 + 32 + lane);
          const int cnt = min(32, n_u - st0);
          for (int j = 0; j < cnt; ++j) load_kv(uf_entry_phys(__shfl_sync(0xffffffffu, mine, j)), h);
        }
        for (int j = 0; j < a.n_sink; ++j) load_kv(j, h);
        for (int j = 0; j < a.n_cur; ++j) load_kv(a.cur_phys0 + j, h);
      UF_ITEM_LOOP_END
    } else if (warp == kW0 + 1 && rank == 0) {
      // ================================ MMA issuer (leader CTA) ======================
      // S(j) = Q K(j)^T for j = 0, 1, 2 up front; then per block n: O += P(n) V(n), S(n+3) = Q K(n+3)^T into buffer n mod 3.
      const uint32_t q_lo = desc_lo(base + kOff2Q, 16);
      const uint32_t k_lo_base = desc_lo(base + kOff2K, 16);
      const uint32_t v_lo_base = desc_lo(base + kOff2V, kHalf);
      uint32_t ks = 0, kph = 0, vs = 0, vph = 0, qph = 0, pph = 0;      // pph: one parity bit per S / P buffer
      uint32_t pv_count = 0;                                            // O += P V launches so far
      auto issue_qk = [&](int buf) {
        mbar_wait(bars + (B2_K_FULL0 + ks) * 8, kph);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t k_lo = k_lo_base + ks * (kHalfTile >> 4);
#pragma unroll
          for (int k = 0; k < 8; ++k)
            // 16 elements = 32 B along K; the second 64-column box is 16 KB further in the Q tile (128 rows), 8 KB in
            // this CTA's K half (64 rows)
            ufptx::mma_ss_2sm(tmem + buf * 128, q_lo + (((k & 3) * 32 + (k >> 2) * kHalf) >> 4),
                              k_lo + (((k & 3) * 32 + (k >> 2) * (kHalfTile / 2)) >> 4), kIdescQK2, k == 0 ? 0u : 1u);
          ufptx::tc_commit_2sm(bars + (B2_S_FULL0 + buf) * 8);
          ufptx::tc_commit_2sm(bars + (B2_K_EMPTY0 + ks) * 8);
        }
        if (++ks == kNK2) { ks = 0; kph ^= 1; }
      };
      UF_ITEM_LOOP_BEGIN
        (void)ulist; (void)full_mask;
        const int n_steps = n_u + a.n_sink + a.n_cur;
        mbar_wait(bars + B2_Q_FULL * 8, qph);
        qph ^= 1;
        for (int j = 0; j < 3 && j < n_steps; ++j) issue_qk(j);
        for (int n = 0, buf = 0; n < n_steps; ++n, buf = (buf == 2 ? 0 : buf + 1)) {
          mbar_wait(bars + (B2_P_FULL0 + buf) * 8, (pph >> buf) & 1u);
          pph ^= 1u << buf;
          mbar_wait(bars + (B2_V_FULL0 + vs) * 8, vph);
          tc_fence_after();
          if (elect_one()) {
            // B = this CTA's V half: 128 keys x 64 columns, MN-major: 16 keys = 2048 B per K step
            const uint32_t v_lo = v_lo_base + vs * (kHalfTile >> 4);
            const uint32_t p_tmem = tmem + buf * 128;
#pragma unroll
            for (int k = 0; k < 8; ++k)
              ufptx::mma_ts_2sm(tmem + 384, p_tmem + (k >> 2) * 64 + (k & 3) * 8, v_lo + k * (2048 >> 4), kDescHi, kIdescPV2,
                                (n == 0 && k == 0) ? 0u : 1u);
            ufptx::tc_commit_2sm(bars + (B2_V_EMPTY0 + vs) * 8);
            ufptx::tc_commit_2sm(bars + (B2_PV_DONE0 + (pv_count & 1u)) * 8);
          }
          ++pv_count;
          if (++vs == kNV2) { vs = 0; vph ^= 1; }
          if (n + 3 < n_steps) issue_qk(buf);
        }
        if (elect_one()) ufptx::tc_commit_2sm(bars + B2_O_FULL * 8);
      UF_ITEM_LOOP_END
    }
  } else if (kGroups == 2) {
    // ============================ softmax + epilogue, two groups of 8 warps (both CTAs) ======================
    // 640 threads x 96 registers at launch; 16 x 32 x 104 + 4 x 32 x 40 fits that pool (112 would not: the request
    // would never be granted)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
    const int grp = warp >> 3;                         // group: takes the steps with global number gs = grp (mod 2)
    const int wq = warp & 3;                           // TMEM lane quarter
    const int half = (warp >> 2) & 1;                  // which 64 keys of a block
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    const uint32_t col0 = (uint32_t)half * 64;
    const float sl2 = a.sl2;
    const uint64_t sl22 = pack2(sl2, sl2);
    volatile uint8_t* xc = reinterpret_cast<volatile uint8_t*>(base_ptr + kOff2Xc);     // [group][half][row][parity]
    volatile uint8_t* x_own = xc + ((grp * 2 + half) * 128 + row) * 2;
    volatile uint8_t* x_oth = xc + ((grp * 2 + (half ^ 1)) * 128 + row) * 2;
    volatile float* m0_s = reinterpret_cast<volatile float*>(base_ptr + kOff2M0);       // [row]
    volatile int* rc_s = reinterpret_cast<volatile int*>(base_ptr + kOff2Rc);           // [row]
    volatile uint32_t* cnt_s = reinterpret_cast<volatile uint32_t*>(base_ptr + kOff2Cnt);
    const uint32_t o_tmem = tmem + lane_addr + 384 + col0;                              // this thread's 64 O columns (rescale)
    uint32_t oph = 0, sph = 0;                         // sph: one parity bit per S buffer, toggled at EVERY step
    uint32_t gs = 0;                                   // global step number (all items, all steps, both groups count)
    auto pow2neg = [](int k) { return __int_as_float((127 - min(k, 126)) << 23); };     // 2^-k

    UF_ITEM_LOOP_BEGIN
      const bool tile_exists = (full_mask >> rank) & 1;
      float m0 = 0.f, l = 0.f;                         // the row's reference max is m0 + r
      int r_loc = 0;                                   // r this thread's l (and last P) is relative to
      int d_own = 0, par = 0, n = 0;
      uint32_t buf = 0;                                // S / P buffer of the step: n mod 3 (the MMA warp restarts at 0 per item)
      bool seen_first = false;                         // a block this tile attends has been processed (by either group)
      bool have_m = false;                             // this thread has taken part since: m0, r_loc, l are valid

      // one key block.  mine: this group's turn.  Every thread of both groups walks all steps (gs, seen_first).
      auto step = [&](const bool attend, const int nvalid) {
        const bool mine = ((gs & 1u) == (uint32_t)grp);
        if (mine) {
          const uint32_t s_tmem = tmem + lane_addr + buf * 128 + col0;      // this thread's 64 S columns
          const int left = nvalid - (int)col0;
          mbar_wait(bars + (B2_S_FULL0 + buf) * 8, (sph >> buf) & 1u);
          tc_fence_after();
          // the previous step (the other group's) has published its decision (its successor on the same barrier, step
          // gs + 1, waits for this step's: no aliasing)
          if (gs > 0u) mbar_wait(bars + (B2_DEC0 + ((gs - 1u) & 1u)) * 8, ((gs - 1u) >> 1) & 1u);
          asm volatile("bar.sync %0, 64;" ::"r"(2 + grp * 4 + wq) : "memory");          // row partners step together
          uint32_t sa[32], pk[16];
          int D_eff = 0;
          const bool exact = attend && !seen_first;
          if (attend && seen_first) {
            // adopt the row's current m; raise it if this group's previous step asked for more
            const int r_cur = rc_s[row];
            const bool joined = have_m;      // else: first block this thread computes in the item (its partner's too)
            if (!joined) { m0 = m0_s[row]; r_loc = r_cur; l = 0.f; have_m = true; d_own = 0; }
            const int want = r_loc + (joined ? max(d_own, (int)x_oth[par ^ 1]) : 0);   // relative to this group's last step
            const int r_new = max(r_cur, want);
            D_eff = r_new - r_cur;
            l *= pow2neg(r_new - r_loc);
            r_loc = r_new;
          }
          asm volatile("bar.sync %0, 64;" ::"r"(2 + grp * 4 + wq) : "memory");          // both threads of the row have read r
          if (D_eff > 0 && half == 0) rc_s[row] = r_loc;
          if (exact) {
            // first attended block of the item: exact row max before the exponentials
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              UF_TMEM_LD32(s_tmem + c * 32, sa, 0);
              UF_TMEM_WAIT_LD32(sa);
#pragma unroll
              for (int u = 0; u < 32; u += 2) {
                const float v0 = (c * 32 + u < left) ? __uint_as_float(sa[u]) : -INFINITY;
                const float v1 = (c * 32 + u + 1 < left) ? __uint_as_float(sa[u + 1]) : -INFINITY;
                if (u & 2) mx1 = max3(mx1, v0, v1); else mx0 = max3(mx0, v0, v1);
              }
            }
            const uint32_t mine_b = bf16_bits_up(fmaxf(mx0, mx1));
            *reinterpret_cast<volatile uint16_t*>(x_own) = (uint16_t)mine_b;
            asm volatile("bar.sync %0, 64;" ::"r"(2 + grp * 4 + wq) : "memory");
            const uint32_t theirs = *reinterpret_cast<volatile uint16_t*>(x_oth);
            asm volatile("bar.sync %0, 64;" ::"r"(2 + grp * 4 + wq) : "memory");
            m0 = fmaxf(__uint_as_float(mine_b << 16), __uint_as_float(theirs << 16)) * sl2;
            r_loc = 0; l = 0.f; have_m = true; d_own = 0;
            x_own[0] = 0; x_own[1] = 0;                 // the exchange slots held the bf16 max: no raise pending
            if (half == 0) { m0_s[row] = m0; rc_s[row] = 0; }
          }
          // publish: everything this step decided is in shared memory before the next step may start
          __threadfence_block();
          asm volatile("bar.sync %0, 256;" ::"r"(10 + grp) : "memory");
          if ((warp & 7) == 0 && lane == 0) mbar_arrive(bars + (B2_DEC0 + (gs & 1u)) * 8);
          int Dnew = 0;
          if (attend) {
            const float m = m0 + (float)r_loc;
            const uint64_t nm2 = pack2(-m, -m);
            uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
            UF_TMEM_LD32(s_tmem + 0, sa, 0);
            UF_TMEM_WAIT_LD32(sa);
            exp_chunk(sa, pk, half * 2 + 0, left, sl22, nm2, acc0, acc1);
            UF_TMEM_ST16(s_tmem + 0, pk);
            UF_TMEM_LD32(s_tmem + 32, sa, 0);
            UF_TMEM_WAIT_LD32(sa);
            exp_chunk(sa, pk, half * 2 + 1, left - 32, sl22, nm2, acc0, acc1);
            UF_TMEM_ST16(s_tmem + 16, pk);
            float a0, a1, b0, b1;
            unpack2(acc0, a0, a1);
            unpack2(acc1, b0, b1);
            const float lsum = (a0 + a1) + (b0 + b1);
            l += lsum;
            if (!(lsum <= 256.0f)) {
              if (lsum < kPanicSum) {
                Dnew = (int)((__float_as_uint(lsum) >> 23) & 0xffu) - 126;
              } else {
                a.panic_item[it] = a.seq;
                *a.panic_last = a.seq;
                Dnew = 101;
              }
            }
          } else {
            // a block only the other tile of the pair attends: P = 0
#pragma unroll
            for (int c = 0; c < 16; ++c) pk[c] = 0u;
            UF_TMEM_ST16(s_tmem + 0, pk);
            UF_TMEM_ST16(s_tmem + 16, pk);
          }
          x_own[par] = (uint8_t)Dnew;
          d_own = Dnew;
          par ^= 1;
          // O still holds the blocks before this one relative to the m before this step's raise: every O += P V issued
          // so far must be complete (the previous step's, number gs - 1, was the last), the next waits for our P_FULL
          if (__any_sync(0xffffffffu, D_eff > 0) && n > 0) {
            const uint32_t g = gs - 1u;
            mbar_wait(bars + (B2_PV_DONE0 + (g & 1u)) * 8, (g >> 1) & 1u);
            tc_fence_after();
            const float f = pow2neg(D_eff);
#pragma unroll
            for (int cc = 0; cc < 64; cc += 32) {
              UF_TMEM_LD32(o_tmem + cc, sa, 0);
              UF_TMEM_WAIT_LD32(sa);
#pragma unroll
              for (int c = 0; c < 32; ++c) sa[c] = __float_as_uint(__uint_as_float(sa[c]) * f);
              UF_TMEM_ST32(o_tmem + cc, sa, 0);
            }
          }
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) ufptx::mbar_arrive_leader(bars + (B2_P_FULL0 + buf) * 8);
        }
        if (attend) seen_first = true;
        sph ^= 1u << buf;
        buf = (buf == 2u) ? 0u : buf + 1u;
        ++gs;
        ++n;
      };

      {
        int32_t mine_e = 0;
        for (int st = 0; st < n_u; ++st) {
          if ((st & 31) == 0) mine_e = (st + lane < n_u) ? __ldg(ulist + st + lane) : 0;
          const int32_t e = __shfl_sync(0xffffffffu, mine_e, st & 31);
          step(((uf_entry_mask(e) >> rank) & 1) != 0, uf_entry_nvalid(e));
        }
        for (int j = 0; j < a.n_sink + a.n_cur; ++j) {
          const int nvalid = (j < a.n_sink) ? min(128, a.sink_ntok - j * 128) : min(128, a.ntok - (j - a.n_sink) * 128);
          step(tile_exists, nvalid);
        }
      }

      // ---- epilogue: O / l -> bf16 -> swizzled staging (the Q buffer) -> TMA store; the 16 warps split O 4 ways ----
      {
        unsigned char* stage = base_ptr + kOff2Q;
        mbar_wait(bars + B2_O_FULL * 8, oph);          // every MMA of the item is complete: Q is free too
        oph ^= 1;
        tc_fence_after();
        asm volatile("bar.sync 1, 512;" ::: "memory");                     // every step's decision is in shared memory
        const int r_fin = have_m ? rc_s[row] : 0;
        volatile float* xl = reinterpret_cast<volatile float*>(stage);
        xl[(grp * 2 + half) * 128 + row] = have_m ? l * pow2neg(r_fin - r_loc) : 0.f;
        asm volatile("bar.sync 1, 512;" ::: "memory");
        const float l_tot = (xl[row] + xl[128 + row]) + (xl[256 + row] + xl[384 + row]);
        const float m_fin = m0_s[row] + (float)rc_s[row];
        asm volatile("bar.sync 1, 512;" ::: "memory");                     // all read before the staging writes
        const float inv = 1.0f / l_tot;
        {
          uint32_t ov[32];
          UF_TMEM_LD32(tmem + lane_addr + 384 + col0 + grp * 32, ov, 0);   // columns [64 half + 32 grp, + 32)
          UF_TMEM_WAIT_LD32(ov);
          unsigned char* half_base = stage + half * kHalf + row * 128;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 w;
            w.x = pack_bf16x2(__uint_as_float(ov[8 * j + 0]) * inv, __uint_as_float(ov[8 * j + 1]) * inv);
            w.y = pack_bf16x2(__uint_as_float(ov[8 * j + 2]) * inv, __uint_as_float(ov[8 * j + 3]) * inv);
            w.z = pack_bf16x2(__uint_as_float(ov[8 * j + 4]) * inv, __uint_as_float(ov[8 * j + 5]) * inv);
            w.w = pack_bf16x2(__uint_as_float(ov[8 * j + 6]) * inv, __uint_as_float(ov[8 * j + 7]) * inv);
            const int chunk = grp * 4 + j;
            *reinterpret_cast<uint4*>(half_base + ((chunk ^ (row & 7)) << 4)) = w;
          }
        }
        tc_fence_before();
        fence_proxy_async();
        asm volatile("bar.sync 1, 512;" ::: "memory");
        const int row0 = (2 * p + rank) * 128;
        if (warp == 0 && lane == 0) {
          if (tile_exists) {
            const uint32_t src = base + kOff2Q;
            tma_store_3d(&tm_o, src, 0, row0, h);
            tma_store_3d(&tm_o, src + kHalf, 64, row0, h);
            tma_store_commit_and_wait_read();
          }
          mbar_arrive(bars + B2_Q_EMPTY * 8);
        }
        if (tile_exists && grp == 0 && half == 0 && a.lse != nullptr && row0 + row < a.ntok)
          a.lse[(int64_t)h * a.ntok + row0 + row] = (m_fin + log2f(l_tot)) * 0.6931471805599453f;
      }
    UF_ITEM_LOOP_END
    if (warp == 0 && lane == 0) tma_store_wait_all();
  } else {
    // ================================== softmax + epilogue (both CTAs) ======================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    const int wq = warp & 3;                           // TMEM lane quarter
    const int half = warp >> 2;                        // which 64 keys of a block / 64 columns of O
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    const uint32_t col0 = (uint32_t)half * 64;
    const float sl2 = a.sl2;
    const uint64_t sl22 = pack2(sl2, sl2);
    volatile uint8_t* xc = reinterpret_cast<volatile uint8_t*>(base_ptr + kOff2Xc);     // [half][row][parity]
    volatile uint8_t* x_own = xc + (half * 128 + row) * 2;
    volatile uint8_t* x_oth = xc + ((half ^ 1) * 128 + row) * 2;
    const uint32_t o_tmem = tmem + lane_addr + 384 + col0;
    uint32_t sph = 0, oph = 0;                         // sph: one parity bit per S buffer
    uint32_t pv_seen = 0;                              // O += P V launches of this CTA pair before the current step

    UF_ITEM_LOOP_BEGIN
      const bool tile_exists = (full_mask >> rank) & 1;
      float m = -INFINITY, l = 0.f;
      int d_own = 0, par = 0, n = 0, buf = 0;
      bool first = true;

      // multiply this thread's half of the O row by f; O must be quiescent: every O += P V issued so far is complete
      // (PV_DONE of the previous step) and the next one waits for this step's P_FULL
      // The tensor pipe may lag the softmax by up to two blocks, so O += P V number g signals PV_DONE[g & 1]: of that
      // barrier's phases the one before ((g - 2): complete, S_FULL of this step was committed after it) and the
      // one waited for are the only candidates, and the parity wait cannot alias.
      auto rescale_o = [&](float f) {
        const uint32_t g = pv_seen - 1;
        mbar_wait(bars + (B2_PV_DONE0 + (g & 1u)) * 8, (g >> 1) & 1u);
        tc_fence_after();
#pragma unroll
        for (int cc = 0; cc < 64; cc += 32) {
          uint32_t ov[32];
          UF_TMEM_LD32(o_tmem + cc, ov, 0);
          UF_TMEM_WAIT_LD32(ov);
#pragma unroll
          for (int c = 0; c < 32; ++c) ov[c] = __float_as_uint(__uint_as_float(ov[c]) * f);
          UF_TMEM_ST32(o_tmem + cc, ov, 0);
        }
      };

      auto softmax_step = [&](const bool attend, const int nvalid) {
        const uint32_t s_tmem = tmem + lane_addr + buf * 128 + col0;       // this thread's 64 S columns
        const int left = nvalid - (int)col0;
        mbar_wait(bars + (B2_S_FULL0 + buf) * 8, (sph >> buf) & 1u);
        sph ^= 1u << buf;
        tc_fence_after();
        // the two threads of a row step together (S_FULL no longer implies that the partner finished the last step)
        asm volatile("bar.sync %0, 64;" ::"r"(2 + wq) : "memory");
        uint32_t sa[32], sb[32], pk[16];
        float f_o = 1.0f;                              // pending factor for O (applied at the end of the step)
        if (!kSafe && !first) {
          const int D = max(d_own, (int)x_oth[par ^ 1]);
          if (D > 0) {
            f_o = __int_as_float((127 - D) << 23);     // 2^-D
            l *= f_o;
            m += (float)D;
          }
        }
        int Dnew = 0;
        if (attend) {
          if (kSafe || first) {
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              UF_TMEM_LD32(s_tmem + c * 32, sa, 0);
              UF_TMEM_WAIT_LD32(sa);
#pragma unroll
              for (int u = 0; u < 32; u += 2) {
                const float v0 = (c * 32 + u < left) ? __uint_as_float(sa[u]) : -INFINITY;
                const float v1 = (c * 32 + u + 1 < left) ? __uint_as_float(sa[u + 1]) : -INFINITY;
                if (u & 2) mx1 = max3(mx1, v0, v1); else mx0 = max3(mx0, v0, v1);
              }
            }
            const uint32_t mine = bf16_bits_up(fmaxf(mx0, mx1));
            *reinterpret_cast<volatile uint16_t*>(x_own) = (uint16_t)mine;
            asm volatile("bar.sync %0, 64;" ::"r"(2 + wq) : "memory");
            const uint32_t theirs = *reinterpret_cast<volatile uint16_t*>(x_oth);
            const float rowmax = fmaxf(__uint_as_float(mine << 16), __uint_as_float(theirs << 16));
            asm volatile("bar.sync %0, 64;" ::"r"(2 + wq) : "memory");
            const float m_new = fmaxf(m, rowmax * sl2);
            if (first) {
              m = m_new;
              first = false;
            } else if ((m_new - m) > kRescaleThreshold) {          // kSafe only
              f_o = ex2(m - m_new);
              m = m_new;
              l *= f_o;
            }
          }
          const uint64_t nm2 = pack2(-m, -m);
          uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
          UF_TMEM_LD32(s_tmem + 0, sa, 0);
          UF_TMEM_WAIT_LD32(sa);
          UF_TMEM_LD32(s_tmem + 32, sb, 0);
          exp_chunk(sa, pk, half * 2 + 0, left, sl22, nm2, acc0, acc1);
          UF_TMEM_ST16(s_tmem + 0, pk);
          UF_TMEM_WAIT_LD32(sb);
          exp_chunk(sb, pk, half * 2 + 1, left - 32, sl22, nm2, acc0, acc1);
          UF_TMEM_ST16(s_tmem + 16, pk);
          float a0, a1, b0, b1;
          unpack2(acc0, a0, a1);
          unpack2(acc1, b0, b1);
          const float lsum = (a0 + a1) + (b0 + b1);
          l += lsum;
          if (!kSafe && !(lsum <= 256.0f)) {
            if (lsum < kPanicSum) {
              Dnew = (int)((__float_as_uint(lsum) >> 23) & 0xffu) - 126;
            } else {
              a.panic_item[it] = a.seq;
              *a.panic_last = a.seq;
              Dnew = 101;
            }
          }
        } else {
          // a block only the other tile of the pair attends: P = 0
#pragma unroll
          for (int c = 0; c < 16; ++c) pk[c] = 0u;
          UF_TMEM_ST16(s_tmem + 0, pk);
          UF_TMEM_ST16(s_tmem + 16, pk);
        }
        if (!kSafe) {
          x_own[par] = (uint8_t)Dnew;
          d_own = Dnew;
        }
        par ^= 1;
        // O still holds the blocks before this one relative to the old m
        if (__any_sync(0xffffffffu, f_o != 1.0f) && n > 0) rescale_o(f_o);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) ufptx::mbar_arrive_leader(bars + (B2_P_FULL0 + buf) * 8);
        ++n;
        buf = (buf == 2) ? 0 : buf + 1;
        ++pv_seen;
      };

      {
        int32_t mine = 0;
        for (int st = 0; st < n_u; ++st) {
          if ((st & 31) == 0) mine = (st + lane < n_u) ? __ldg(ulist + st + lane) : 0;
          const int32_t e = __shfl_sync(0xffffffffu, mine, st & 31);
          softmax_step(((uf_entry_mask(e) >> rank) & 1) != 0, uf_entry_nvalid(e));
        }
        for (int j = 0; j < a.n_sink + a.n_cur; ++j) {
          const int nvalid = (j < a.n_sink) ? min(128, a.sink_ntok - j * 128) : min(128, a.ntok - (j - a.n_sink) * 128);
          softmax_step(tile_exists, nvalid);
        }
      }

      // ---- epilogue: O / l -> bf16 -> swizzled staging (the Q buffer) -> TMA store ----
      {
        unsigned char* stage = base_ptr + kOff2Q;
        mbar_wait(bars + B2_O_FULL * 8, oph);          // every MMA of the item is complete: Q is free too
        oph ^= 1;
        tc_fence_after();
        volatile float* xl = reinterpret_cast<volatile float*>(stage);
        xl[half * 128 + row] = l;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const float l_tot = l + xl[(half ^ 1) * 128 + row];
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const float inv = 1.0f / l_tot;
#pragma unroll
        for (int cc = 0; cc < 64; cc += 32) {
          uint32_t ov[32];
          UF_TMEM_LD32(o_tmem + cc, ov, 0);
          UF_TMEM_WAIT_LD32(ov);
          unsigned char* half_base = stage + half * kHalf + row * 128;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 w;
            w.x = pack_bf16x2(__uint_as_float(ov[8 * j + 0]) * inv, __uint_as_float(ov[8 * j + 1]) * inv);
            w.y = pack_bf16x2(__uint_as_float(ov[8 * j + 2]) * inv, __uint_as_float(ov[8 * j + 3]) * inv);
            w.z = pack_bf16x2(__uint_as_float(ov[8 * j + 4]) * inv, __uint_as_float(ov[8 * j + 5]) * inv);
            w.w = pack_bf16x2(__uint_as_float(ov[8 * j + 6]) * inv, __uint_as_float(ov[8 * j + 7]) * inv);
            const int chunk = (cc >> 3) + j;
            *reinterpret_cast<uint4*>(half_base + ((chunk ^ (row & 7)) << 4)) = w;
          }
        }
        tc_fence_before();
        fence_proxy_async();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const int row0 = (2 * p + rank) * 128;
        if (warp == 0 && lane == 0) {
          if (tile_exists) {
            const uint32_t src = base + kOff2Q;
            tma_store_3d(&tm_o, src, 0, row0, h);
            tma_store_3d(&tm_o, src + kHalf, 64, row0, h);
            tma_store_commit_and_wait_read();
          }
          mbar_arrive(bars + B2_Q_EMPTY * 8);
        }
        if (tile_exists && half == 0 && a.lse != nullptr && row0 + row < a.ntok)
          a.lse[(int64_t)h * a.ntok + row0 + row] = (m + log2f(l_tot)) * 0.6931471805599453f;
      }
    UF_ITEM_LOOP_END
    if (warp == 0 && lane == 0) tma_store_wait_all();
  }
#undef UF_ITEM_LOOP_BEGIN
#undef UF_ITEM_LOOP_END

  tc_fence_before();
  __syncthreads();
  ufptx::cluster_sync();                               // neither CTA frees TMEM or exits while the other may still use it
  if (warp == kW0 + 2) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
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
bool encode_map(CUtensorMap* m, const void* ptr, uint64_t rows, uint64_t H, uint64_t row_stride, uint64_t head_stride,
                uint32_t box_rows = 128) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[3] = {128, rows, H};
  const cuuint64_t strides[2] = {row_stride * 2, head_stride * 2};
  const cuuint32_t box[3] = {64, box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Q / O maps are looked up in the ctx's small cache first (a tensor map is a pure function of the key)
const CUtensorMap* cached_map(uf_ctx* c, const void* ptr, int rows, int H, int64_t tok_stride, int64_t head_stride) {
  for (int i = 0; i < c->tm_cache_n; ++i) {
    const uf_ctx::TmEntry& e = c->tm_cache[i];
    if (e.ptr == ptr && e.rows == rows && e.tok_stride == tok_stride && e.head_stride == head_stride) return &e.map;
  }
  uf_ctx::TmEntry& e = c->tm_cache[c->tm_cache_next];
  if (!encode_map(&e.map, ptr, rows, H, tok_stride, head_stride)) { e.ptr = nullptr; return nullptr; }
  e.ptr = ptr; e.rows = rows; e.tok_stride = tok_stride; e.head_stride = head_stride;
  c->tm_cache_next = (c->tm_cache_next + 1) % uf_ctx::kTmCache;
  if (c->tm_cache_n < uf_ctx::kTmCache) ++c->tm_cache_n;
  return &e.map;
}

}  // namespace

int uf_sm100_make_cache_maps(uf_ctx* c) {
  const uint64_t rows = (uint64_t)c->P * 128;
  if (!encode_map(&c->tm_k, c->kc, rows, c->cfg.n_heads, 128, rows * 128) ||
      !encode_map(&c->tm_k_half, c->kc, rows, c->cfg.n_heads, 128, rows * 128, 64) ||
      !encode_map(&c->tm_v, c->vc, rows, c->cfg.n_heads, 128, rows * 128)) {
    c->err = "cuTensorMapEncodeTiled failed for the K/V cache";
    return UF_ERR_CUDA;
  }
  cudaError_t e = cudaFuncSetAttribute(uf_attn_sm100_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(uf_attn_sm100_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(uf_attn_pair_kernel<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes2);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(uf_attn_pair_kernel<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes2);
  if (e != cudaSuccess) {
    c->err = std::string("cudaFuncSetAttribute(smem): ") + cudaGetErrorString(e);
    return UF_ERR_CUDA;
  }
  c->tm_ok = true;
  return UF_OK;
}

int uf_launch_attn_sm100(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, __nv_bfloat16* o, float* lse,
                         int64_t tok_stride, int64_t head_stride, float scale, cudaStream_t s) {
  // each map is copied before the next lookup: a miss may recycle the very cache entry the previous hit returned
  const CUtensorMap* pq = cached_map(c, q, v.cur_ntok, v.H, tok_stride, head_stride);
  if (!pq) {
    c->err = "cuTensorMapEncodeTiled failed for Q (check strides and alignment)";
    return UF_ERR_INVALID_ARG;
  }
  const CUtensorMap tm_q = *pq;
  const CUtensorMap* po = cached_map(c, o, v.cur_ntok, v.H, tok_stride, head_stride);
  if (!po) {
    c->err = "cuTensorMapEncodeTiled failed for O (check strides and alignment)";
    return UF_ERR_INVALID_ARG;
  }
  const CUtensorMap tm_o = *po;
  AttnParams a;
  a.sel_pair = c->sel_pair; a.pair_cnt = c->pair_cnt; a.lse = lse;
  a.H = v.H; a.NP = (v.BPC + 1) / 2; a.kcap = c->kcap;
  a.ntok = v.cur_ntok; a.nqb = uf_ceil_div(v.cur_ntok, 128); a.np_cur = (a.nqb + 1) / 2;
  a.n_sink = v.n_sink_blocks; a.sink_ntok = v.sink_ntok;
  a.n_cur = c->sel_paper ? 0 : a.nqb;
  a.cur_phys0 = v.S + v.cur_slot * v.BPC;
  a.sl2 = scale * 1.4426950408889634f;
  const int n_items = a.H * a.np_cur;
  const int grid = n_items < c->sm_count ? n_items : c->sm_count;
  if (++c->attn_seq <= 0) c->attn_seq = 1;
  a.panic_item = c->panic_item; a.panic_last = c->panic_last; a.seq = c->attn_seq;
  // fast kernel, then the safe kernel for the items it flagged (returns at once when there are none)
  if (c->attn_impl == 2) {
    // CTA pairs: one query tile per CTA, the pair shares every K / V tile, two softmax groups per CTA (640 threads);
    // flagged items are redone by the one-group exact-max instantiation
    const int pairs = n_items < c->sm_count / 2 ? n_items : c->sm_count / 2;
    uf_attn_pair_kernel<false, 2><<<2 * pairs, 20 * 32, kSmemBytes2, s>>>(tm_q, tm_o, c->tm_k_half, c->tm_v, a);
    uf_attn_pair_kernel<true, 1><<<2 * pairs, kThreads, kSmemBytes2, s>>>(tm_q, tm_o, c->tm_k_half, c->tm_v, a);
  } else {
    uf_attn_sm100_kernel<false><<<grid, kThreads, kSmemBytes, s>>>(tm_q, tm_o, c->tm_k, c->tm_v, a);
    uf_attn_sm100_kernel<true><<<grid, kThreads, kSmemBytes, s>>>(tm_q, tm_o, c->tm_k, c->tm_v, a);
  }
  c->launches += 2;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    c->err = std::string("uf_attn_sm100_kernel launch: ") + cudaGetErrorString(e);
    return UF_ERR_CUDA;
  }
  return UF_OK;
}
