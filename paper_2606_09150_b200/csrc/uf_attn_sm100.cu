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

namespace {

constexpr int kNK = 3;                 // K ring stages
constexpr int kNV = 2;                 // V ring stages
constexpr int kTile = 128 * 128 * 2;   // bytes of one 128 x 128 bf16 tile
constexpr int kHalf = kTile / 2;       // one 64-column box
constexpr int kThreads = 384;
constexpr float kRescaleThreshold = 8.0f;   // log2 units

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

__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
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

// shared-memory matrix descriptor, 128-byte swizzle
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
         (1ull << 46) | (2ull << 61);
}

// instruction descriptor kind::f16: D fp32, A/B bf16, M = N = 128; B MN-major for P V
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescQK | (1u << 16);

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

__device__ __forceinline__ Item get_item(const AttnParams& a, int it) {
  Item x;
  x.h = it / a.np_cur;
  x.p = it % a.np_cur;
  const int64_t pi = (int64_t)x.h * a.NP + x.p;
  x.n_u = a.pair_cnt[pi];
  x.ulist = a.sel_pair + pi * 2 * a.kcap;
  x.n_steps = x.n_u + a.n_sink + a.nqb;
  x.full_mask = (2 * x.p + 1 < a.nqb) ? 3 : 1;
  return x;
}

__device__ __forceinline__ int32_t get_entry(const AttnParams& a, const Item& x, int st) {
  if (st < x.n_u) return __ldg(x.ulist + st);
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
      mbar_init(bars + i * 8, softmax_arrives ? 128u : 1u);
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

  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    if (warp == 8 && lane == 0) {
      // ================================ TMA producer ================================
      uint32_t kcount = 0, vcount = 0, qn[2] = {0, 0};
      for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item x = get_item(a, it);
        for (int t = 0; t < 2; ++t) {
          if (!(x.full_mask & (1 << t))) continue;
          const uint32_t bq = bars + (Q_FULL0 + t) * 8;
          mbar_wait(bars + (Q_EMPTY0 + t) * 8, (qn[t] & 1) ^ 1);
          mbar_expect_tx(bq, kTile);
          const int row0 = (2 * x.p + t) * 128;
          tma_load_3d(base + kOffQ + t * kTile, &tm_q, bq, 0, row0, x.h);
          tma_load_3d(base + kOffQ + t * kTile + kHalf, &tm_q, bq, 64, row0, x.h);
          ++qn[t];
        }
        int32_t e = get_entry(a, x, 0);
        for (int st = 0; st < x.n_steps; ++st) {
          const int32_t en = (st + 1 < x.n_steps) ? get_entry(a, x, st + 1) : 0;
          const int row = uf_entry_phys(e) * 128;
          {
            const uint32_t s = kcount % kNK, n = kcount / kNK;
            const uint32_t bf = bars + (K_FULL0 + s) * 8;
            mbar_wait(bars + (K_EMPTY0 + s) * 8, (n & 1) ^ 1);
            mbar_expect_tx(bf, kTile);
            tma_load_3d(base + kOffK + s * kTile, &tm_k, bf, 0, row, x.h);
            tma_load_3d(base + kOffK + s * kTile + kHalf, &tm_k, bf, 64, row, x.h);
            ++kcount;
          }
          {
            const uint32_t s = vcount % kNV, n = vcount / kNV;
            const uint32_t bf = bars + (V_FULL0 + s) * 8;
            mbar_wait(bars + (V_EMPTY0 + s) * 8, (n & 1) ^ 1);
            mbar_expect_tx(bf, kTile);
            tma_load_3d(base + kOffV + s * kTile, &tm_v, bf, 0, row, x.h);
            tma_load_3d(base + kOffV + s * kTile + kHalf, &tm_v, bf, 64, row, x.h);
            ++vcount;
          }
          e = en;
        }
      }
    } else if (warp == 9 && lane == 0) {
      // ================================ MMA issuer ==================================
      uint32_t kcount = 0, vcount = 0, qn[2] = {0, 0}, pn[2] = {0, 0};
      int vrem[kNV];
#pragma unroll
      for (int i = 0; i < kNV; ++i) vrem[i] = 0;
      for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item x = get_item(a, it);
        bool pend[2] = {false, false};
        uint32_t pend_vs[2] = {0, 0}, pend_vpar[2] = {0, 0};
        bool first_pv[2] = {true, true};
        for (int t = 0; t < 2; ++t)
          if (x.full_mask & (1 << t)) { mbar_wait(bars + (Q_FULL0 + t) * 8, qn[t] & 1); ++qn[t]; }

        auto do_pv = [&](int t) {
          mbar_wait(bars + (P_FULL0 + t) * 8, pn[t] & 1); ++pn[t];
          const uint32_t vs = pend_vs[t];
          mbar_wait(bars + (V_FULL0 + vs) * 8, pend_vpar[t]);
          tc_fence_after();
          const uint32_t vaddr = base + kOffV + vs * kTile;
          const uint32_t d_tmem = tmem + 256 + t * 128;
          const uint32_t p_tmem = tmem + t * 128;
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            // B = V tile, MN-major: 8-key groups 1024 B apart (SBO), the two 64-column halves 16 KB apart (LBO)
            const uint64_t bd = make_desc(vaddr + k * 2048, kHalf, 1024);
            mma_ts(d_tmem, p_tmem + k * 8, bd, kIdescPV, (first_pv[t] && k == 0) ? 0u : 1u);
          }
          first_pv[t] = false;
          if (--vrem[vs] == 0) tc_commit(bars + (V_EMPTY0 + vs) * 8);
          pend[t] = false;
        };

        int32_t e = get_entry(a, x, 0);
        for (int st = 0; st < x.n_steps; ++st) {
          const int32_t en = (st + 1 < x.n_steps) ? get_entry(a, x, st + 1) : 0;
          const int m = uf_entry_mask(e);
          const uint32_t ks = kcount % kNK, kpar = (kcount / kNK) & 1;
          const uint32_t vs = vcount % kNV, vpar = (vcount / kNV) & 1;
          mbar_wait(bars + (K_FULL0 + ks) * 8, kpar);
          tc_fence_after();
          const uint32_t kaddr = base + kOffK + ks * kTile;
          int users = 0;
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            if (!(m & (1 << t))) continue;
            if (pend[t]) do_pv(t);
            const uint32_t qaddr = base + kOffQ + t * kTile;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              // K-major operands: 8-row groups 1024 B apart (SBO); 16 elements = 32 B along K, second half +16 KB
              const uint32_t koff = (k & 3) * 32 + (k >> 2) * kHalf;
              mma_ss(tmem + t * 128, make_desc(qaddr + koff, 16, 1024), make_desc(kaddr + koff, 16, 1024), kIdescQK,
                     k == 0 ? 0u : 1u);
            }
            tc_commit(bars + (S_FULL0 + t) * 8);
            pend[t] = true; pend_vs[t] = vs; pend_vpar[t] = vpar;
            ++users;
          }
          tc_commit(bars + (K_EMPTY0 + ks) * 8);
          vrem[vs] = users;
          ++kcount; ++vcount;
#pragma unroll
          for (int t = 0; t < 2; ++t)
            if (!(m & (1 << t)) && pend[t]) do_pv(t);      // keep V stages flowing (no deadlock)
          e = en;
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (pend[t]) do_pv(t);
          if (x.full_mask & (1 << t)) tc_commit(bars + (O_FULL0 + t) * 8);
        }
      }
    }
  } else {
    // ================================== softmax + epilogue ==================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
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
        mbar_wait(b_sfull, sn & 1); ++sn;
        tc_fence_after();
        uint32_t s[128];
        UF_TMEM_LD32(s_tmem + 0, s, 0);
        UF_TMEM_LD32(s_tmem + 32, s, 32);
        UF_TMEM_LD32(s_tmem + 64, s, 64);
        UF_TMEM_LD32(s_tmem + 96, s, 96);
        tmem_wait_ld();
        if (nvalid < 128) {
#pragma unroll
          for (int c = 0; c < 128; ++c)
            if (c >= nvalid) s[c] = 0xff800000u;       // -inf: ragged key block (R-3)
        }
        float mx0 = __uint_as_float(s[0]), mx1 = __uint_as_float(s[1]), mx2 = __uint_as_float(s[2]), mx3 = __uint_as_float(s[3]);
#pragma unroll
        for (int c = 4; c < 128; c += 4) {
          mx0 = fmaxf(mx0, __uint_as_float(s[c]));
          mx1 = fmaxf(mx1, __uint_as_float(s[c + 1]));
          mx2 = fmaxf(mx2, __uint_as_float(s[c + 2]));
          mx3 = fmaxf(mx3, __uint_as_float(s[c + 3]));
        }
        const float m_new = fmaxf(m, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * a.sl2);
        if (first) {
          m = m_new;
          first = false;
        } else {
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
          }
        }
        float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
        uint32_t pk[64];
#pragma unroll
        for (int c = 0; c < 128; c += 4) {
          const float p0 = ex2(fmaf(__uint_as_float(s[c]), a.sl2, -m));
          const float p1 = ex2(fmaf(__uint_as_float(s[c + 1]), a.sl2, -m));
          const float p2 = ex2(fmaf(__uint_as_float(s[c + 2]), a.sl2, -m));
          const float p3 = ex2(fmaf(__uint_as_float(s[c + 3]), a.sl2, -m));
          l0 += p0; l1 += p1; l2 += p2; l3 += p3;
          pk[c / 2] = pack_bf16x2(p0, p1);
          pk[c / 2 + 1] = pack_bf16x2(p2, p3);
        }
        l += (l0 + l1) + (l2 + l3);
        UF_TMEM_ST32(s_tmem + 0, pk, 0);
        UF_TMEM_ST32(s_tmem + 32, pk, 32);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(b_pfull);
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
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    c->err = std::string("uf_attn_sm100_kernel launch: ") + cudaGetErrorString(e);
    return UF_ERR_CUDA;
  }
  return UF_OK;
}
