// uf_fused_append.cu — SURVEY 8(f) NEXT-2: everything that touches Q, K, V before the attention, in ONE pass over the
// QKV projection output (Wan2.1 architecture, "3D RoPE with axis dims (44,42,42)"; readings R-37..R-40):
//   QK-norm (RMS over the token's whole hidden vector, learned weight) -> 3-D RoPE -> bf16
//   -> post-RoPE Q to the caller's buffer + block-mean pooled Q (so uf_select_blocks has nothing left to pool)
//   -> post-RoPE K and V into the cache slot (step a1) + block-mean pooled K.
// HBM traffic: Q, K, V read once, Q', K-cache, V-cache written once (6 * N*H*d*2 bytes); the second look at Q, K
// inside the CTA comes from L1/L2.
//
// Arithmetic (R-40): bf16 -> fp64, every operation IEEE fp64 rounded once, no FMA contraction, in the order
//   ss = sum x^2;  r = 1 / sqrt(ss / C + eps);  u = (x * r) * g;  out_e = u_e*cos - u_o*sin;  out_o = u_e*sin + u_o*cos
// then ONE rounding fp64 -> bf16 (nearest even, below 2^-126 -> signed zero), done on the bits, which also yields
// the rounded value as a double for the pooled sums (exact, order-free, as in uf_append.cu).  This makes the cache
// bytes and the pooled means a fixed function of the input bits: the oracle (oracle/uf_rope_norm.py) gets the same.
//
// One CTA per key block of the chunk (all heads).  Phase 1, token-major: one warp per token row streams the row's
// H*d channels of Q and K (16-byte vectors, coalesced) and reduces the two sums of squares -> r_q[row], r_k[row] in
// shared memory.  Phase 2, column-major per head (the layout of uf_append_kernel): thread = (16-byte column, row
// group); it owns 4 RoPE pairs whose axis (t / y / x) is fixed, so it reads one cos/sin pair per (row, RoPE pair) from
// the fp64 tables (model state, L1/L2 resident), and keeps the pooled sums of its 8 channels in registers.
#include "uf_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ uint4 ld_keep(const uint4* p) { return __ldg(p); }

__device__ __forceinline__ double bf16lo(uint32_t w) { return (double)__uint_as_float(w << 16); }
__device__ __forceinline__ double bf16hi(uint32_t w) { return (double)__uint_as_float(w & 0xFFFF0000u); }

// fp64 -> bf16, round to nearest even on the bits (R-40): returns the bf16 bits and, through *rounded, the rounded
// value as a double.  keep = exponent (11 bits) + top 7 mantissa bits; the 45 bits below decide the rounding; a carry
// into the exponent is the right result.  Magnitudes below 2^-126 after rounding become signed zero.
__device__ __forceinline__ uint32_t round_bf16(double y, double* rounded) {
  const uint32_t hi = (uint32_t)__double2hiint(y), lo = (uint32_t)__double2loint(y);
  const uint32_t sign = hi & 0x80000000u, mag = hi & 0x7FFFFFFFu;
  uint32_t keep = mag >> 13;
  const uint32_t rest = mag & 0x1FFFu;
  const bool up = rest > 0x1000u || (rest == 0x1000u && (lo != 0u || (keep & 1u)));
  keep += up ? 1u : 0u;
  const uint32_t bias = (1023u - 127u) << 7;
  const bool small = keep < bias + 128u;
  *rounded = small ? __hiloint2double((int)sign, 0) : __hiloint2double((int)(sign | (keep << 13)), 0);
  return (sign >> 16) | (small ? 0u : keep - bias);
}

struct FusedParams {
  const __nv_bfloat16 *q, *k, *v;
  __nv_bfloat16* q_out;
  int64_t in_ts, in_hs, out_ts, out_hs;
  const double *cos_tab, *sin_tab;     // [max_pos][D/2]
  const float *gq, *gk;                // [H*D]
  double eps;
  int t0, Hg, Wg;                      // raster mode: token n -> (t0 + n / (Hg*Wg), (n / Wg) % Hg, n % Wg)
  int pairs_t, pairs_th;               // RoPE pair p: p < pairs_t -> t, p < pairs_th -> y, else x
  __nv_bfloat16 *kc, *vc;
  double *kpool, *qbar;
  int H, B, P, BPC, ntok, phys0, sink_copy_blocks;
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

template <int D>
__global__ void __launch_bounds__(kThreads)
uf_fused_append_kernel(const FusedParams a) {
  constexpr int VPR = D / 8;                 // 16-byte vectors per head row
  constexpr int RPP = kThreads / VPR;        // row groups
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* r_q = reinterpret_cast<double*>(smem_raw);           // [B]
  double* r_k = r_q + a.B;                                     // [B]
  int* pos_s = reinterpret_cast<int*>(r_k + a.B);              // [B][3]
  double* red = reinterpret_cast<double*>(pos_s + 3 * a.B + (a.B & 1));   // [2][RPP][D + 2]
  const int b = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row0 = b * a.B;
  const int nvalid = a.til.enabled ? uf_tile_nvalid(a.til, b) : min(a.B, a.ntok - row0);
  const int C = a.H * D;
  const int VT = C / 8;                      // vectors per token row

  // ---- phase 1: RMS factors of the block's rows (R-37), token-major --------------------------------------------
  for (int r = warp; r < nvalid; r += kWarps) {
    const int64_t base = (int64_t)(row0 + r) * a.in_ts;
    double sq = 0.0, sk = 0.0;
    for (int v = lane; v < VT; v += 32) {
      const int h = v / VPR, c8 = (v % VPR) * 8;
      const int64_t off = base + (int64_t)h * a.in_hs + c8;
      const uint4 uq = ld_keep(reinterpret_cast<const uint4*>(a.q + off));
      const uint4 uk = ld_keep(reinterpret_cast<const uint4*>(a.k + off));
      const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const double q0 = bf16lo(wq[i]), q1 = bf16hi(wq[i]), k0 = bf16lo(wk[i]), k1 = bf16hi(wk[i]);
        sq = fma(q0, q0, sq); sq = fma(q1, q1, sq);          // x*x is exact in fp64: fma == mul then add
        sk = fma(k0, k0, sk); sk = fma(k1, k1, sk);
      }
    }
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) {
      sq = __dadd_rn(sq, __shfl_xor_sync(0xffffffffu, sq, sh));
      sk = __dadd_rn(sk, __shfl_xor_sync(0xffffffffu, sk, sh));
    }
    if (lane == 0) {
      r_q[r] = __ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sq, (double)C), a.eps)));
      r_k[r] = __ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sk, (double)C), a.eps)));
      int t, y, x;
      row_pos(a, b, r, &t, &y, &x);
      pos_s[3 * r] = t; pos_s[3 * r + 1] = y; pos_s[3 * r + 2] = x;
    }
  }
  __syncthreads();

  // ---- phase 2: per head, column-major: norm * weight, RoPE, round, write, pool --------------------------------
  const int vcx = tid % VPR, rg = tid / VPR;
  const int phys = a.phys0 + b;
  const bool to_sink = b < a.sink_copy_blocks;
  // this thread's 4 RoPE pairs p = vcx*4 + j and the axis each one follows
  int axis[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int p = vcx * 4 + j;
    axis[j] = p < a.pairs_t ? 0 : (p < a.pairs_th ? 1 : 2);
  }
  const uint4 zero = make_uint4(0, 0, 0, 0);
  for (int h = 0; h < a.H; ++h) {
    double gqv[8], gkv[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      gqv[e] = (double)__ldg(a.gq + h * D + vcx * 8 + e);
      gkv[e] = (double)__ldg(a.gk + h * D + vcx * 8 + e);
    }
    double pq[8], pk[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { pq[e] = 0.0; pk[e] = 0.0; }
    const int64_t dst = (((int64_t)h * a.P + phys) * a.B) * D;
    const int64_t dst_sink = (((int64_t)h * a.P + b) * a.B) * D;
    for (int r = rg; r < a.B; r += RPP) {
      uint4 oq = zero, ok = zero, ov = zero;
      if (r < nvalid) {
        const int64_t src = (int64_t)(row0 + r) * a.in_ts + (int64_t)h * a.in_hs + vcx * 8;
        const uint4 uq = ld_keep(reinterpret_cast<const uint4*>(a.q + src));     // second read: L1 / L2
        const uint4 uk = ld_keep(reinterpret_cast<const uint4*>(a.k + src));
        ov = ld_stream(reinterpret_cast<const uint4*>(a.v + src));
        const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
        uint32_t rq[4], rk[4];
        const double rq_f = r_q[r], rk_f = r_k[r];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int pos = pos_s[3 * r + axis[j]];
          const int64_t ti = (int64_t)pos * (D / 2) + vcx * 4 + j;
          const double cs = __ldg(a.cos_tab + ti), sn = __ldg(a.sin_tab + ti);
          // q
          {
            const double ue = __dmul_rn(__dmul_rn(bf16lo(wq[j]), rq_f), gqv[2 * j]);
            const double uo = __dmul_rn(__dmul_rn(bf16hi(wq[j]), rq_f), gqv[2 * j + 1]);
            const double oe = __dsub_rn(__dmul_rn(ue, cs), __dmul_rn(uo, sn));
            const double oo = __dadd_rn(__dmul_rn(ue, sn), __dmul_rn(uo, cs));
            double re, ro;
            const uint32_t be = round_bf16(oe, &re), bo = round_bf16(oo, &ro);
            rq[j] = be | (bo << 16);
            pq[2 * j] += re; pq[2 * j + 1] += ro;
          }
          // k
          {
            const double ue = __dmul_rn(__dmul_rn(bf16lo(wk[j]), rk_f), gkv[2 * j]);
            const double uo = __dmul_rn(__dmul_rn(bf16hi(wk[j]), rk_f), gkv[2 * j + 1]);
            const double oe = __dsub_rn(__dmul_rn(ue, cs), __dmul_rn(uo, sn));
            const double oo = __dadd_rn(__dmul_rn(ue, sn), __dmul_rn(uo, cs));
            double re, ro;
            const uint32_t be = round_bf16(oe, &re), bo = round_bf16(oo, &ro);
            rk[j] = be | (bo << 16);
            pk[2 * j] += re; pk[2 * j + 1] += ro;
          }
        }
        oq = make_uint4(rq[0], rq[1], rq[2], rq[3]);
        ok = make_uint4(rk[0], rk[1], rk[2], rk[3]);
      }
      // rows past nvalid are written as zeros (pad rows of ragged blocks / tiles)
      const int64_t o = (int64_t)r * D + vcx * 8;
      *reinterpret_cast<uint4*>(a.kc + dst + o) = ok;
      *reinterpret_cast<uint4*>(a.vc + dst + o) = ov;
      if (to_sink) {
        *reinterpret_cast<uint4*>(a.kc + dst_sink + o) = ok;
        *reinterpret_cast<uint4*>(a.vc + dst_sink + o) = ov;
      }
      if (r < nvalid || a.til.enabled)      // raster mode: rows past the chunk's end do not exist in q_out
        *reinterpret_cast<uint4*>(a.q_out + (int64_t)(row0 + r) * a.out_ts + (int64_t)h * a.out_hs + vcx * 8) = oq;
    }
    // block sums of this head: reduce the row groups through shared memory (exact sums: order-free)
    double* redq = red;
    double* redk = red + RPP * (D + 2);
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      redq[rg * (D + 2) + vcx * 8 + e] = pq[e];
      redk[rg * (D + 2) + vcx * 8 + e] = pk[e];
    }
    __syncthreads();
    if (tid < 2 * D) {
      const int col = tid % D;
      const double* src = tid < D ? redq : redk;
      double s = 0.0;
#pragma unroll
      for (int g = 0; g < RPP; ++g) s += src[g * (D + 2) + col];
      const double mean = s / (double)nvalid;               // mean over the valid rows only (R-3)
      if (tid < D) {
        a.qbar[((int64_t)h * a.BPC + b) * D + col] = mean;
      } else {
        a.kpool[((int64_t)h * D + col) * a.P + phys] = mean;
        if (to_sink) a.kpool[((int64_t)h * D + col) * a.P + b] = mean;
      }
    }
    __syncthreads();
  }
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
  const size_t smem = (size_t)2 * v.B * 8 + (size_t)(3 * v.B + (v.B & 1)) * 4 + (size_t)2 * (kThreads / (D / 8)) * (D + 2) * 8;
  uf_fused_append_kernel<D><<<nb, kThreads, smem, s>>>(a);
  c->launches += 1;
  return cudaGetLastError();
}
