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
// and the oracle (oracle/uf_rope_norm.py) does the same in NumPy float32.  The pooled sums add the ROUNDED values in
// fp64 (exact, order-free, as in uf_append.cu).
//
// Grid: a thread-block CLUSTER per key block of the chunk; the CS CTAs of a cluster split the heads (CS = the largest
// divisor of H that is <= 8).  Phase 1, token-major: one warp per token row streams its CTA's heads of Q and K (16-byte
// vectors, coalesced) and reduces the partial sums of squares; the partials of the CS CTAs are combined through
// distributed shared memory (rank order) into r_q[row], r_k[row].  Phase 2, column-major per head (the layout of
// uf_append_kernel): thread = (16-byte column, row group); it owns 4 RoPE pairs whose axis (t / y / x) is fixed, reads
// one cos / sin pair per (row, RoPE pair) from the fp32 tables (model state, L1/L2 resident) and keeps the pooled sums
// of its 8 channels in registers.  The second look at Q, K comes from L1 / L2.
#include "uf_internal.h"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

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
  int CS, HPC;                         // CTAs per cluster, heads per CTA (CS * HPC == H)
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
  double* part_q = reinterpret_cast<double*>(smem_raw);        // [B] this CTA's partial sums of squares (own heads)
  double* part_k = part_q + a.B;                               // [B]
  float* r_q = reinterpret_cast<float*>(part_k + a.B);         // [B]
  float* r_k = r_q + a.B;                                      // [B]
  int* pos_s = reinterpret_cast<int*>(r_k + a.B);              // [B][3]
  double* red = reinterpret_cast<double*>(pos_s + 3 * a.B + (a.B & 1));   // [2][RPP][D + 2]
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int b = blockIdx.x / a.CS;
  const int h0 = rank * a.HPC;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row0 = b * a.B;
  const int nvalid = a.til.enabled ? uf_tile_nvalid(a.til, b) : min(a.B, a.ntok - row0);
  const int C = a.H * D;
  const int VT = a.HPC * VPR;                // vectors of this CTA's heads per token row

  // ---- phase 1: partial sums of squares of this CTA's heads (R-37), token-major --------------------------------
  for (int r = warp; r < nvalid; r += kWarps) {
    const int64_t base = (int64_t)(row0 + r) * a.in_ts;
    double sq = 0.0, sk = 0.0;
    for (int v = lane; v < VT; v += 32) {
      const int h = h0 + v / VPR, c8 = (v % VPR) * 8;
      const int64_t off = base + (int64_t)h * a.in_hs + c8;
      const uint4 uq = ld_keep(reinterpret_cast<const uint4*>(a.q + off));
      const uint4 uk = ld_keep(reinterpret_cast<const uint4*>(a.k + off));
      const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float q0 = bf16lo(wq[i]), q1 = bf16hi(wq[i]), k0 = bf16lo(wk[i]), k1 = bf16hi(wk[i]);
        // x*x is exact in fp32 (8 x 8 significant bits); the sum runs in fp64 (exact)
        sq += (double)__fmul_rn(q0, q0); sq += (double)__fmul_rn(q1, q1);
        sk += (double)__fmul_rn(k0, k0); sk += (double)__fmul_rn(k1, k1);
      }
    }
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) {
      sq = __dadd_rn(sq, __shfl_xor_sync(0xffffffffu, sq, sh));
      sk = __dadd_rn(sk, __shfl_xor_sync(0xffffffffu, sk, sh));
    }
    if (lane == 0) {
      part_q[r] = sq; part_k[r] = sk;
      int t, y, x;
      row_pos(a, b, r, &t, &y, &x);
      pos_s[3 * r] = t; pos_s[3 * r + 1] = y; pos_s[3 * r + 2] = x;
    }
  }
  cluster.sync();                            // every CTA's partials are visible cluster-wide
  if (tid < nvalid) {
    double sq = 0.0, sk = 0.0;
    for (int k = 0; k < a.CS; ++k) {         // rank order (the sums are exact, so any order gives the same bits)
      const double* rq = cluster.map_shared_rank(part_q, k);
      const double* rk = cluster.map_shared_rank(part_k, k);
      sq = __dadd_rn(sq, rq[tid]);
      sk = __dadd_rn(sk, rk[tid]);
    }
    r_q[tid] = __double2float_rn(__ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sq, (double)C), a.eps))));
    r_k[tid] = __double2float_rn(__ddiv_rn(1.0, __dsqrt_rn(__dadd_rn(__ddiv_rn(sk, (double)C), a.eps))));
  }
  cluster.sync();                            // remote reads are done before any CTA moves on / exits

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
  for (int h = h0; h < h0 + a.HPC; ++h) {
    float gqv[8], gkv[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      gqv[e] = __ldg(a.gq + h * D + vcx * 8 + e);
      gkv[e] = __ldg(a.gk + h * D + vcx * 8 + e);
    }
    double pq[8], pk[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { pq[e] = 0.0; pk[e] = 0.0; }
    const int64_t dst = (((int64_t)h * a.P + phys) * a.B) * D;
    const int64_t dst_sink = (((int64_t)h * a.P + b) * a.B) * D;
#pragma unroll 2
    for (int r = rg; r < a.B; r += RPP) {
      uint4 oq = zero, ok = zero, ov = zero;
      if (r < nvalid) {
        const int64_t src = (int64_t)(row0 + r) * a.in_ts + (int64_t)h * a.in_hs + vcx * 8;
        const uint4 uq = ld_keep(reinterpret_cast<const uint4*>(a.q + src));     // second read: L1 / L2
        const uint4 uk = ld_keep(reinterpret_cast<const uint4*>(a.k + src));
        ov = ld_stream(reinterpret_cast<const uint4*>(a.v + src));
        const uint32_t wq[4] = {uq.x, uq.y, uq.z, uq.w}, wk[4] = {uk.x, uk.y, uk.z, uk.w};
        uint32_t rq[4], rk[4];
        const float rq_f = r_q[r], rk_f = r_k[r];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int pos = pos_s[3 * r + axis[j]];
          const int64_t ti = (int64_t)pos * (D / 2) + vcx * 4 + j;
          const float cs = __ldg(a.cos_tab + ti), sn = __ldg(a.sin_tab + ti);
          {
            const float ue = __fmul_rn(__fmul_rn(bf16lo(wq[j]), rq_f), gqv[2 * j]);
            const float uo = __fmul_rn(__fmul_rn(bf16hi(wq[j]), rq_f), gqv[2 * j + 1]);
            const float oe = __fsub_rn(__fmul_rn(ue, cs), __fmul_rn(uo, sn));
            const float oo = __fadd_rn(__fmul_rn(ue, sn), __fmul_rn(uo, cs));
            const uint32_t w = pack_bf16x2(oe, oo);
            rq[j] = w;
            pq[2 * j] += (double)bf16lo(w); pq[2 * j + 1] += (double)bf16hi(w);   // the ROUNDED values (exact sums)
          }
          {
            const float ue = __fmul_rn(__fmul_rn(bf16lo(wk[j]), rk_f), gkv[2 * j]);
            const float uo = __fmul_rn(__fmul_rn(bf16hi(wk[j]), rk_f), gkv[2 * j + 1]);
            const float oe = __fsub_rn(__fmul_rn(ue, cs), __fmul_rn(uo, sn));
            const float oo = __fadd_rn(__fmul_rn(ue, sn), __fmul_rn(uo, cs));
            const uint32_t w = pack_bf16x2(oe, oo);
            rk[j] = w;
            pk[2 * j] += (double)bf16lo(w); pk[2 * j + 1] += (double)bf16hi(w);
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
  int cs = 1;
  for (int k = 8; k >= 1; --k) if (v.H % k == 0) { cs = k; break; }   // largest divisor of H that fits a portable cluster
  a.CS = cs; a.HPC = v.H / cs;
  const size_t smem = (size_t)2 * v.B * 8 + (size_t)2 * v.B * 4 + (size_t)(3 * v.B + (v.B & 1)) * 4 +
                      (size_t)2 * (kThreads / (D / 8)) * (D + 2) * 8;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(nb * cs));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  cudaError_t e = cudaLaunchKernelEx(&cfg, uf_fused_append_kernel<D>, a);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}
