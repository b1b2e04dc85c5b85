// uf_append.cu — step a1: write one chunk's K,V into the cache slot chosen by the host policy and
// produce the block-mean pooled K of each of its blocks.  HBM-bound: every K,V byte is read
// once and written once with 16-byte vector accesses; the pooled sums ride along in fp64 (a sum of
// <= 128 bf16 values is exact in fp64, so the result does not depend on the summation order, R-4).
#include "uf_internal.h"

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

__device__ __forceinline__ void acc_bf16x8(double* acc, const uint4& u) {
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    acc[2 * i]     += (double)__uint_as_float(w[i] << 16);
    acc[2 * i + 1] += (double)__uint_as_float(w[i] & 0xFFFF0000u);
  }
}

// grid (blocks of the chunk, H); each CTA moves one B x d tile of K and of V.
// Thread t: vector column vc = t % (d/8), row group rg = t / (d/8); rows rg, rg+RPP, ...
template <int D>
__global__ void __launch_bounds__(kThreads)
uf_append_kernel(const __nv_bfloat16* __restrict__ k, const __nv_bfloat16* __restrict__ v,
                 int64_t tok_stride, int64_t head_stride,
                 __nv_bfloat16* __restrict__ kc, __nv_bfloat16* __restrict__ vc, double* __restrict__ kpool,
                 int B, int P, int ntok, int phys0, int sink_copy_blocks, UfTiling til) {
  constexpr int VPR = D / 8;               // 16-byte vectors per row
  constexpr int RPP = kThreads / VPR;      // rows per pass
  __shared__ double red[RPP][D + 2];
  const int b = blockIdx.x, h = blockIdx.y;
  const int vcx = threadIdx.x % VPR, rg = threadIdx.x / VPR;
  const int row0 = b * B;
  const int nvalid = til.enabled ? uf_tile_nvalid(til, b) : min(B, ntok - row0);   // tiled: rows [0, nvalid) of the block
  const int phys = phys0 + b;
  const bool to_sink = b < sink_copy_blocks;          // chunk 0: blocks 0..S-1 also go to the sink region
  const int64_t dst = (((int64_t)h * P + phys) * B) * D;
  const int64_t dst_sink = (((int64_t)h * P + b) * B) * D;
  double acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.0;
  const uint4 zero = make_uint4(0, 0, 0, 0);
#pragma unroll 4
  for (int r = rg; r < B; r += RPP) {
    uint4 kk = zero, vv = zero;
    if (r < nvalid) {
      const int64_t src = (int64_t)(row0 + r) * tok_stride + (int64_t)h * head_stride + vcx * 8;
      kk = ld_stream(reinterpret_cast<const uint4*>(k + src));
      vv = ld_stream(reinterpret_cast<const uint4*>(v + src));
      acc_bf16x8(acc, kk);
    }
    // rows past nvalid are written as zeros: the attention kernel relies on zero V padding
    const int64_t o = (int64_t)r * D + vcx * 8;
    *reinterpret_cast<uint4*>(kc + dst + o) = kk;
    *reinterpret_cast<uint4*>(vc + dst + o) = vv;
    if (to_sink) {
      *reinterpret_cast<uint4*>(kc + dst_sink + o) = kk;
      *reinterpret_cast<uint4*>(vc + dst_sink + o) = vv;
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) red[rg][vcx * 8 + i] = acc[i];
  __syncthreads();
  if (threadIdx.x < D) {
    double s = 0.0;
#pragma unroll
    for (int g = 0; g < RPP; ++g) s += red[g][threadIdx.x];
    const double mean = s / (double)nvalid;            // mean over the valid rows only (R-3)
    kpool[((int64_t)h * D + threadIdx.x) * P + phys] = mean;
    if (to_sink) kpool[((int64_t)h * D + threadIdx.x) * P + b] = mean;
  }
}

// ---- raster <-> tiled token order (paper-mask mode, R-29) ------------------------------------------
// One warp per (tiled row, head).  Tiled row R = b*B + r holds, for r < nvalid(b), the r-th token of tile b in
// raster order inside the tile; rows r >= nvalid(b) are pad (written as zeros when tiling, skipped when untiling).
constexpr int kTileWarps = 8;
__global__ void __launch_bounds__(kTileWarps * 32)
uf_tile_kernel(const __nv_bfloat16* __restrict__ src, __nv_bfloat16* __restrict__ dst, int64_t src_ts, int64_t src_hs,
               int64_t dst_ts, int64_t dst_hs, UfTiling til, int B, int H, int d, int n_rows, bool untile) {
  const int lane = threadIdx.x & 31;
  const int64_t wid = (int64_t)blockIdx.x * kTileWarps + (threadIdx.x >> 5);
  if (wid >= (int64_t)n_rows * H) return;
  const int R = (int)(wid / H), h = (int)(wid % H);
  const int b = R / B, r = R % B;
  int it, ih, iw;
  uf_tile_coords(til, b, &it, &ih, &iw);
  const int vh = min(til.bh, til.Hg - ih * til.bh), vw = min(til.bw, til.Wg - iw * til.bw);
  const int nvalid = uf_tile_nvalid(til, b);
  const int words = d / 2;
  if (r >= nvalid) {
    if (!untile) {
      uint32_t* o = reinterpret_cast<uint32_t*>(dst + (int64_t)R * dst_ts + (int64_t)h * dst_hs);
      for (int w = lane; w < words; w += 32) o[w] = 0u;
    }
    return;
  }
  const int dt = r / (vh * vw), dy = (r / vw) % vh, dx = r % vw;
  const int64_t n = ((int64_t)(it * til.bt + dt) * til.Hg + (ih * til.bh + dy)) * til.Wg + (iw * til.bw + dx);
  const int64_t tiled_off = (int64_t)R, raster_off = n;
  const uint32_t* in = reinterpret_cast<const uint32_t*>(
      src + (untile ? tiled_off : raster_off) * src_ts + (int64_t)h * src_hs);
  uint32_t* out = reinterpret_cast<uint32_t*>(dst + (untile ? raster_off : tiled_off) * dst_ts + (int64_t)h * dst_hs);
  for (int w = lane; w < words; w += 32) out[w] = in[w];
}

}  // namespace

cudaError_t uf_launch_tile(uf_ctx* c, const __nv_bfloat16* src, __nv_bfloat16* dst, int64_t src_tok_stride,
                           int64_t src_head_stride, int64_t dst_tok_stride, int64_t dst_head_stride, bool untile,
                           cudaStream_t s) {
  const UfTiling& t = c->til;
  const int n_rows = t.nbt * t.nbh * t.nbw * c->cfg.block;
  const int64_t warps = (int64_t)n_rows * c->cfg.n_heads;
  uf_tile_kernel<<<(unsigned)((warps + kTileWarps - 1) / kTileWarps), kTileWarps * 32, 0, s>>>(
      src, dst, src_tok_stride, src_head_stride, dst_tok_stride, dst_head_stride, t, c->cfg.block, c->cfg.n_heads,
      c->cfg.head_dim, n_rows, untile);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t uf_launch_append(uf_ctx* c, const UfView& v, const __nv_bfloat16* k, const __nv_bfloat16* vv,
                             int64_t tok_stride, int64_t head_stride, cudaStream_t s) {
  const int nb = uf_ceil_div(v.cur_ntok, v.B);
  dim3 grid(nb, v.H);
  const int phys0 = v.S + v.cur_slot * v.BPC;
  const int sink_copy = v.cur_chunk == 0 ? min(uf_ceil_div(v.sink_ntok, v.B), nb) : 0;
#define UF_APPEND_CASE(DD)                                                                              \
  case DD:                                                                                              \
    uf_append_kernel<DD><<<grid, kThreads, 0, s>>>(k, vv, tok_stride, head_stride, c->kc, c->vc,        \
                                                   c->kpool, v.B, v.P, v.cur_ntok, phys0, sink_copy,    \
                                                   v.til);                                              \
    break;
  switch (v.d) {
    UF_APPEND_CASE(32)
    UF_APPEND_CASE(64)
    UF_APPEND_CASE(128)
    default: return cudaErrorInvalidValue;
  }
#undef UF_APPEND_CASE
  c->launches += 1;
  return cudaGetLastError();
}
