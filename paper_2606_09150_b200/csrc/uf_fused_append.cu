// uf_fused_append.cu — SURVEY 8(f) NEXT-2: everything that touches Q, K, V before the attention, in ONE pass over the
// QKV projection output (Wan2.1 architecture, "3D RoPE with axis dims (44,42,42)"; readings R-37..R-40):
//   QK-norm (RMS over the token's whole hidden vector, learned weight) -> 3-D RoPE -> bf16
//   -> post-RoPE Q to the caller's buffer + block-mean pooled Q (so uf_select_blocks has nothing left to pool)
//   -> post-RoPE K and V into the cache slot (step a1) + block-mean pooled K.
// HBM traffic: Q, K, V read once, Q', K-cache, V-cache written once (6 * N*H*d*2 bytes); the second look at Q, K
// inside the CTA comes from L1/L2.
//
// Arithmetic (R-40): the bf16 rounding of the result decides cache bytes and (through pooling) block indices, so it is
// taken on a number that is a fixed function of the input bits: IEEE fp32, every operation rounded once, no FMA
// contraction (__fmul_rn / __fadd_rn / __fsub_rn), in the order
//   ss = sum x^2 (fp64, exact);  r = fl32(1 / sqrt(ss / C + eps)) (fp64 ops);  u = fl(fl(x r) g);
//   out_e = fl(fl(u_e cos) - fl(u_o sin));  out_o = fl(fl(u_e sin) + fl(u_o cos));  result = bf16_rne(out)
// (tests/fused_fp32_model.py restates this order in NumPy float32 for a reproducibility test; the ORACLE,
// oracle/uf_rope_norm.py, is the fp64 definition with one rounding, and the kernel is compared with it within one bf16
// ulp).  The pooled sums add the ROUNDED values in
// fp64 (exact, order-free, as in uf_append.cu).
//
// Grid: a CLUSTER of 8 CTAs per key block of the chunk; each CTA owns B/8 consecutive rows of the block and ALL heads
// (the RMS factor needs a token's whole hidden vector).  The rows go through shared memory in double-buffered batches of
// R rows (cp.async: batch i+1 is in flight while batch i is processed; HBM is read exactly once):
//   phase 1 sum of squares from smem: F2F.F64.BF16 + DFMA per element (x*x is exact, so the fp64 sum is), (row, part)
//           tasks spread over the warps, warp reduce -> r_q, r_k (fp32) in smem;
//   phase 2 thread = one 16-byte column of one head (H * 16 threads): it keeps the norm weights of its 8 channels and the
//           pooled sums of its 8 + 8 channels in REGISTERS and walks the rows: norm, RoPE, round, write Q', K-cache,
//           V-cache, add the rounded values (F2F.F64.BF16 straight from the packed result) to the pooled sums.
// The 8 partial pooled sums of a (head, channel) are combined through distributed shared memory (exact sums: any order
// gives the same bits), divided by the block's valid rows and written to the pooled-K table / pooled-Q buffer.
#include "uf_internal.h"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace {

constexpr int kCluster = 8;             // CTAs per key block
#ifndef UF_FUSED_MINB
#define UF_FUSED_MINB 4
#endif
#ifndef UF_FUSED_STAGE_KB
#define UF_FUSED_STAGE_KB 40
#endif

__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

struct FusedParams {
  const __nv_bfloat16 *q, *k, *v;
  __nv_bfloat16* q_out;
  int64_t in_ts, in_hs, out_ts, out_hs;
  const float *cos_tab, *sin_tab;      // [max_pos][D/2]
  const float *gq, *gk;                // [H*D]
  double eps;
  int t0, Hg, Wg;                      // raster mode: token n -> (t0 + n / (Hg*Wg), (n / Wg) % Hg, n % Wg)
  int pairs_t, pairs_th;               // RoPE pair p: p < pairs_t -> t, p < pairs_th -> y, else x
  __nv_bfloat16 *kc, *vc;
  double *kpool, *qbar;
  int H, B, P, BPC, ntok, phys0, sink_copy_blocks;
  int R, parts;                        // rows per batch (B / 8 is a multiple of it); phase-1 tasks per row
  UfTiling til;
};

// position (t, y, x) of row r of block b
__device__ __forceinline__ void row_pos(const FusedParams& a, int b, int r, int* t, int* y, int* x) {
  if (a.til.enabled) {
    int it, ih, iw;
    uf_tile_coords(a.til, b, &it, &ih, &iw);
    const int vh = min(a.til.bh, a.til.Hg - ih * a.til.bh), vw = min(a.til.bw, a.til.Wg - iw * a.til.bw);
    *t = a.t0 + it * a.til.bt + r / (vh * vw);
    *y = ih * a.til.bh + (r / vw) % vh;
    *x = iw * a.til.bw + r % vw;
  } else {
    const int n = b * a.B + r, per = a.Hg * a.Wg;
    *t = a.t0 + n / per;
    *y = (n % per) / a.Wg;
    *x = n % a.Wg;
  }
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
// bf16 halves of a packed word straight to fp64 (F2F.F64.BF16 with a half-register select: no unpacking)
__device__ __forceinline__ void bf16x2_to_f64(uint32_t w, double* lo, double* hi) {
  unsigned short l, h;
  asm("mov.b32 {%0, %1}, %2;" : "=h"(l), "=h"(h) : "r"(w));
  asm("cvt.f64.bf16 %0, %1;" : "=d"(*lo) : "h"(l));
  asm("cvt.f64.bf16 %0, %1;" : "=d"(*hi) : "h"(h));
}

// HT, RT, PT: compile-time H, rows per batch, phase-1 parts per row (0, 0, 0: taken from the parameters at run time);
// with constants every index computation below folds and the small loops unroll.
template <int D, int kMaxThreads, int kMinBlocks, int HT, int RT, int PT>
__global__ void __launch_bounds__(kMaxThreads, kMinBlocks) uf_fused_append_kernel(const FusedParams a) {
  constexpr int VPR = D / 8;                 // 16-byte vectors per head row
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int H = HT ? HT : a.H;
  const int VT = H * VPR;                    // vectors per token row == worker threads of the CTA
  const int R = RT ? RT : a.R, PARTS = PT ? PT : a.parts;
  const size_t stage_vecs = (size_t)3 * R * VT;                // q, k, v rows of one stage
  uint4* stage_base = reinterpret_cast<uint4*>(smem_raw);      // [2][3][R][VT]
  float2* cs_base = reinterpret_cast<float2*>(stage_base + 2 * stage_vecs);   // [2][R][D/2] (cos, sin)
  float2* rr_s = cs_base + 2 * R * (D / 2);                    // [R] (r_q, r_k)
  double* part_s = reinterpret_cast<double*>(rr_s + R + (R & 1));   // [R][PARTS][2]
  int* pos_all = reinterpret_cast<int*>(part_s + (size_t)R * PARTS * 2);      // [rows_cta][3]
  double* psum = reinterpret_cast<double*>(smem_raw);          // [2][H*D], aliases the stages after the last batch
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int b = blockIdx.x / kCluster;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  const int row0 = b * a.B;
  const int nvalid = a.til.enabled ? uf_tile_nvalid(a.til, b) : min(a.B, a.ntok - row0);
  const int C = H * D;
  const int rows_cta = a.B / kCluster;
  const int rbase = rank * rows_cta;         // first row (inside the block) of this CTA
  const int h = tid / VPR, vcx = tid % VPR;  // this thread's head and 16-byte column (phase 2)
  const bool worker = tid < VT;
  const int phys = a.phys0 + b;
  const bool to_sink = b < a.sink_copy_blocks;
  const int nbatch = rows_cta / R;

  if (tid < rows_cta && rbase + tid < nvalid) {
    int t, y, x;
    row_pos(a, b, rbase + tid, &t, &y, &x);
    pos_all[3 * tid] = t; pos_all[3 * tid + 1] = y; pos_all[3 * tid + 2] = x;
  }
  float gqv[8], gkv[8];
  double pq[8], pk[8];
#pragma unroll
  for (int e = 0; e < 8; ++e) { pq[e] = 0.0; pk[e] = 0.0; gqv[e] = 0.f; gkv[e] = 0.f; }
  if (worker) {
    const float4 g0 = __ldg(reinterpret_cast<const float4*>(a.gq + h * D + vcx * 8));
    const float4 g1 = __ldg(reinterpret_cast<const float4*>(a.gq + h * D + vcx * 8 + 4));
    const float4 g2 = __ldg(reinterpret_cast<const float4*>(a.gk + h * D + vcx * 8));
    const float4 g3 = __ldg(reinterpret_cast<const float4*>(a.gk + h * D + vcx * 8 + 4));
    gqv[0] = g0.x; gqv[1] = g0.y; gqv[2] = g0.z; gqv[3] = g0.w; gqv[4] = g1.x; gqv[5] = g1.y; gqv[6] = g1.z; gqv[7] = g1.w;
    gkv[0] = g2.x; gkv[1] = g2.y; gkv[2] = g2.z; gkv[3] = g2.w; gkv[4] = g3.x; gkv[5] = g3.y; gkv[6] = g3.z; gkv[7] = g3.w;
  }
  const int64_t dst = (((int64_t)h * a.P + phys) * a.B) * D + vcx * 8;
  const int64_t dst_sink = (((int64_t)h * a.P + b) * a.B) * D + vcx * 8;
  const int64_t in_col = (int64_t)h * a.in_hs + vcx * 8;
  const uint4 zero = make_uint4(0, 0, 0, 0);
  __syncthreads();                           // pos_all

  // stage the Q, K, V rows of batch `ib` (the thread's own column of every row) and the rows' cos / sin pairs
  auto issue = [&](int ib) {
    const int st = ib & 1, rb = rbase + ib * R;
    uint4* qs = stage_base + st * stage_vecs;
    if (worker) {
      for (int r = 0; r < R; ++r) {
        if (rb + r >= nvalid) break;
        const int64_t off = (int64_t)(row0 + rb + r) * a.in_ts + in_col;
        cp_async16(qs + (size_t)r * VT + tid, a.q + off);
        cp_async16(qs + (size_t)(R + r) * VT + tid, a.k + off);
        cp_async16(qs + (size_t)(2 * R + r) * VT + tid, a.v + off);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    float2* cs = cs_base + st * R * (D / 2);
    for (int x = tid; x < R * (D / 2); x += blockDim.x) {
      const int r = x / (D / 2), p = x % (D / 2);
      if (rb + r >= nvalid) continue;
      const int* ps = pos_all + 3 * (ib * R + r);
      const int pos = p < a.pairs_t ? ps[0] : (p < a.pairs_th ? ps[1] : ps[2]);
      const int64_t ti = (int64_t)pos * (D / 2) + p;
      cs[x] = make_float2(__ldg(a.cos_tab + ti), __ldg(a.sin_tab + ti));
    }
  };

  issue(0);
  for (int ib = 0; ib < nbatch; ++ib) {
    const int st = ib & 1, rb = rbase + ib * R;
    const int nv_b = max(0, min(R, nvalid - rb));            // valid rows of this batch
    if (ib + 1 < nbatch) {
      issue(ib + 1);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    const uint4* q_s = stage_base + st * stage_vecs;
    const uint4* k_s = q_s + (size_t)R * VT;
    const uint4* v_s = k_s + (size_t)R * VT;
    const float2* cs_s = cs_base + st * R * (D / 2);
    // ---- phase 1: sums of squares (R-37): (row, part) tasks over the warps, fp64 (exact) ----
    const int vpp = (VT + PARTS - 1) / PARTS;                // vectors per part
    for (int task = warp; task < nv_b * PARTS; task += nwarps) {
      const int r = task / PARTS, part = task % PARTS;
      double sq = 0.0, sk = 0.0;
      const int vend = min(VT, (part + 1) * vpp);
#pragma unroll 2
      for (int v = part * vpp + lane; v < vend; v += 32) {
        const uint4 uq = q_s[(size_t)r * VT + v], uk = k_s[(size_t)r * VT + v];
        const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          double q0, q1, k0, k1;
          bf16x2_to_f64(wq[i], &q0, &q1);
          bf16x2_to_f64(wk[i], &k0, &k1);
          sq = fma(q0, q0, sq); sq = fma(q1, q1, sq);          // x*x is exact in fp64: fma == mul then add
          sk = fma(k0, k0, sk); sk = fma(k1, k1, sk);
        }
      }
#pragma unroll
      for (int sh = 16; sh > 0; sh >>= 1) {
        sq = __dadd_rn(sq, __shfl_xor_sync(0xffffffffu, sq, sh));
        sk = __dadd_rn(sk, __shfl_xor_sync(0xffffffffu, sk, sh));
      }
      if (lane == 0) { part_s[(r * PARTS + part) * 2] = sq; part_s[(r * PARTS + part) * 2 + 1] = sk; }
    }
    __syncthreads();
    if (tid < nv_b) {
      double sq = 0.0, sk = 0.0;
      for (int p2 = 0; p2 < PARTS; ++p2) {
        sq = __dadd_rn(sq, part_s[(tid * PARTS + p2) * 2]);
        sk = __dadd_rn(sk, part_s[(tid * PARTS + p2) * 2 + 1]);
      }
      rr_s[tid] = make_float2(
          __double2float_rn(__ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sq, (double)C), a.eps)))),
          __double2float_rn(__ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sk, (double)C), a.eps)))));
    }
    __syncthreads();
    // ---- phase 2: norm * weight, RoPE, round, write, pool ----
    if (worker) {
#pragma unroll 2
      for (int r = 0; r < R; ++r) {
        const int row = rb + r;                               // row inside the block
        uint4 oq = zero, ok = zero, ov = zero;
        if (r < nv_b) {
          const uint4 uq = q_s[(size_t)r * VT + tid], uk = k_s[(size_t)r * VT + tid];
          ov = v_s[(size_t)r * VT + tid];
          const float4 c01 = *reinterpret_cast<const float4*>(cs_s + r * (D / 2) + vcx * 4);       // pairs 0, 1
          const float4 c23 = *reinterpret_cast<const float4*>(cs_s + r * (D / 2) + vcx * 4 + 2);   // pairs 2, 3
          const float csv[4] = {c01.x, c01.z, c23.x, c23.z}, snv[4] = {c01.y, c01.w, c23.y, c23.w};
          const float2 rr = rr_s[r];
          const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
          uint32_t rq[4], rk[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float cs = csv[j], sn = snv[j];
            {
              const float ue = __fmul_rn(__fmul_rn(bf16lo(wq[j]), rr.x), gqv[2 * j]);
              const float uo = __fmul_rn(__fmul_rn(bf16hi(wq[j]), rr.x), gqv[2 * j + 1]);
              const float oe = __fsub_rn(__fmul_rn(ue, cs), __fmul_rn(uo, sn));
              const float oo = __fadd_rn(__fmul_rn(ue, sn), __fmul_rn(uo, cs));
              const uint32_t w = pack_bf16x2(oe, oo);
              rq[j] = w;
              double de, dn;
              bf16x2_to_f64(w, &de, &dn);                     // the ROUNDED values (exact sums)
              pq[2 * j] += de; pq[2 * j + 1] += dn;
            }
            {
              const float ue = __fmul_rn(__fmul_rn(bf16lo(wk[j]), rr.y), gkv[2 * j]);
              const float uo = __fmul_rn(__fmul_rn(bf16hi(wk[j]), rr.y), gkv[2 * j + 1]);
              const float oe = __fsub_rn(__fmul_rn(ue, cs), __fmul_rn(uo, sn));
              const float oo = __fadd_rn(__fmul_rn(ue, sn), __fmul_rn(uo, cs));
              const uint32_t w = pack_bf16x2(oe, oo);
              rk[j] = w;
              double de, dn;
              bf16x2_to_f64(w, &de, &dn);
              pk[2 * j] += de; pk[2 * j + 1] += dn;
            }
          }
          oq = make_uint4(rq[0], rq[1], rq[2], rq[3]);
          ok = make_uint4(rk[0], rk[1], rk[2], rk[3]);
        }
        // rows past nvalid are written as zeros (pad rows of ragged blocks / tiles)
        const int64_t o = (int64_t)row * D;
        *reinterpret_cast<uint4*>(a.kc + dst + o) = ok;
        *reinterpret_cast<uint4*>(a.vc + dst + o) = ov;
        if (to_sink) {
          *reinterpret_cast<uint4*>(a.kc + dst_sink + o) = ok;
          *reinterpret_cast<uint4*>(a.vc + dst_sink + o) = ov;
        }
        if (r < nv_b || a.til.enabled)      // raster mode: rows past the chunk's end do not exist in q_out
          *reinterpret_cast<uint4*>(a.q_out + (int64_t)(row0 + row) * a.out_ts + (int64_t)h * a.out_hs + vcx * 8) = oq;
      }
    }
    __syncthreads();                         // this stage is free for batch ib + 2 (or for psum)
  }

  // ---- pooled means: combine the 8 CTAs' partial sums through distributed shared memory ----
  if (worker) {
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      psum[tid * 8 + e] = pq[e];
      psum[C + tid * 8 + e] = pk[e];
    }
  }
  cluster.sync();
  const int per = (2 * C) / kCluster;        // (tensor, head, channel) entries this CTA finalises
  for (int x = tid; x < per; x += blockDim.x) {
    const int gidx = rank * per + x;         // [2][C]
    double s = 0.0;
    for (int k = 0; k < kCluster; ++k) s = __dadd_rn(s, cluster.map_shared_rank(psum, k)[gidx]);
    const double mean = s / (double)nvalid;                  // mean over the valid rows only (R-3)
    const int isk = gidx / C, ch = gidx % C, hh = ch / D, col = ch % D;
    if (!isk) {
      a.qbar[((int64_t)hh * a.BPC + b) * D + col] = mean;
    } else {
      a.kpool[((int64_t)hh * D + col) * a.P + phys] = mean;
      if (to_sink) a.kpool[((int64_t)hh * D + col) * a.P + b] = mean;
    }
  }
  cluster.sync();                            // nobody leaves while its shared memory is still being read
}

}  // namespace

cudaError_t uf_launch_fused_append(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, const __nv_bfloat16* k,
                                   const __nv_bfloat16* vv, __nv_bfloat16* q_out, int64_t in_ts, int64_t in_hs,
                                   int64_t out_ts, int64_t out_hs, const uf_rope_spec* rs, cudaStream_t s) {
  if (v.d != 128) return cudaErrorInvalidValue;               // RoPE layout (44, 42, 42) is for head_dim 128
  FusedParams a;
  a.q = q; a.k = k; a.v = vv; a.q_out = q_out;
  a.in_ts = in_ts; a.in_hs = in_hs; a.out_ts = out_ts; a.out_hs = out_hs;
  a.cos_tab = rs->cos_tab; a.sin_tab = rs->sin_tab; a.gq = rs->gq; a.gk = rs->gk; a.eps = rs->eps;
  a.t0 = rs->t0; a.Hg = rs->grid_h; a.Wg = rs->grid_w;
  a.pairs_t = rs->dim_t / 2; a.pairs_th = (rs->dim_t + rs->dim_h) / 2;
  a.kc = c->kc; a.vc = c->vc; a.kpool = c->kpool; a.qbar = c->qbar;
  a.H = v.H; a.B = v.B; a.P = v.P; a.BPC = v.BPC; a.ntok = v.cur_ntok;
  a.phys0 = v.S + v.cur_slot * v.BPC;
  const int nb = uf_ceil_div(v.cur_ntok, v.B);
  a.sink_copy_blocks = v.cur_chunk == 0 ? min(uf_ceil_div(v.sink_ntok, v.B), nb) : 0;
  a.til = v.til;
  constexpr int D = 128;
  if (v.B % (kCluster * 2) != 0 || v.B / kCluster > 16 || v.H * (D / 8) > 1024) return cudaErrorInvalidConfiguration;
  const int VT = v.H * (D / 8);
  const int rows_cta = v.B / kCluster;
  const int threads = ((VT + 31) / 32) * 32, nwarps = threads / 32;
  // rows per batch: two stages of Q + K + V rows within ~72 KB (three CTAs per SM at H = 12), and enough for psum
  int R = rows_cta;
  while (R > 1 && (size_t)2 * 3 * R * VT * 16 > UF_FUSED_STAGE_KB * 1024) R >>= 1;
  const size_t psum_bytes = (size_t)2 * v.H * D * 8;
  while (R < rows_cta && (size_t)2 * 3 * R * VT * 16 < psum_bytes) R <<= 1;
  if (rows_cta % R != 0) return cudaErrorInvalidConfiguration;
  auto gcd = [](int x, int y) { while (y) { int t = x % y; x = y; y = t; } return x; };
  a.R = R;
  a.parts = nwarps / gcd(R, nwarps);        // R * parts is a multiple of the warp count: balanced phase 1
  size_t smem = (size_t)2 * 3 * R * VT * 16 + (size_t)2 * R * (D / 2) * 8 + (size_t)(R + (R & 1)) * 8 +
                (size_t)R * a.parts * 2 * 8 + (size_t)rows_cta * 3 * 4;
  if (smem < psum_bytes) smem = psum_bytes;
  // specialised instantiations for the head counts of BASELINE.json (12, 40); anything else takes the generic one
  typedef void (*KernelFn)(const FusedParams);
  KernelFn kern;
  int small;
  if (v.H == 12 && R == 2 && a.parts == 3) { kern = uf_fused_append_kernel<D, 192, UF_FUSED_MINB, 12, 2, 3>; small = 0; }
  else if (v.H == 40 && R == 2 && a.parts == 10) { kern = uf_fused_append_kernel<D, 640, 1, 40, 2, 10>; small = 1; }
  else if (threads <= 256) { kern = uf_fused_append_kernel<D, 256, 3, 0, 0, 0>; small = 2; }
  else { kern = uf_fused_append_kernel<D, 1024, 1, 0, 0, 0>; small = 3; }
  // the limit is a per-device attribute and a ctx lives on one device: the record is kept in the ctx (a ctx is
  // not thread-safe, so neither is this)
  if (smem > 48 * 1024 && smem > c->fused_smem_attr[small]) {
    cudaError_t e0 = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e0 != cudaSuccess) return e0;
    c->fused_smem_attr[small] = smem;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(nb * kCluster));
  cfg.blockDim = dim3((unsigned)threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kCluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  cudaError_t e = cudaLaunchKernelEx(&cfg, kern, a);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}
