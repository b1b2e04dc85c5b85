// uf_attn_generic.cu — step a5 for shapes the tcgen05 kernel does not cover (B != 128 or d != 128,
// e.g. BJ configs[0]: block 64, head_dim 64) and an in-library cross-check of it (uf_set_attn_impl).
// Plain CUDA cores: one warp per query row, lanes split head_dim, online softmax in fp32 over the
// kept key blocks SINK u TOPK[h,i] u CUR in that order (R-13/R-14/R-15).
#include "uf_internal.h"

namespace {

constexpr int kWarps = 8;

template <int D>
__global__ void __launch_bounds__(kWarps * 32)
uf_attn_generic_kernel(UfView v, const __nv_bfloat16* __restrict__ q, __nv_bfloat16* __restrict__ o,
                       float* __restrict__ lse, int64_t tok_stride, int64_t head_stride,
                       const __nv_bfloat16* __restrict__ kc, const __nv_bfloat16* __restrict__ vc,
                       const int32_t* __restrict__ sel_q, const int32_t* __restrict__ sel_cnt, int kcap, int k_eff,
                       float scale) {
  constexpr int EPL = D / 32;                 // elements per lane
  const int i = blockIdx.x, h = blockIdx.y;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int B = v.B;
  const int nqb = uf_ceil_div(v.cur_ntok, B);
  const int rows = min(B, v.cur_ntok - i * B);
  const float sl2 = scale * 1.4426950408889634f;      // logits are handled in the log2 domain
  const int32_t* list = sel_q + ((int64_t)h * v.BPC + i) * kcap;
  // paper-mask mode (sel_cnt != null): only the row's own list (its length in sel_cnt), no SINK, no implicit CUR
  if (sel_cnt) k_eff = sel_cnt[(int64_t)h * v.BPC + i];
  const int n_sink = sel_cnt ? 0 : v.n_sink_blocks;
  const int n_steps = n_sink + k_eff + (sel_cnt ? 0 : nqb);
  const int64_t head_base = (int64_t)h * v.P * B * D;

  for (int r = w; r < rows; r += kWarps) {
    const int64_t qoff = (int64_t)(i * B + r) * tok_stride + (int64_t)h * head_stride + lane * EPL;
    float qv[EPL], acc[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) { qv[e] = __bfloat162float(q[qoff + e]); acc[e] = 0.f; }
    float m = -INFINITY, l = 0.f;
    for (int st = 0; st < n_steps; ++st) {
      int phys, nvalid;
      if (st < n_sink) {                                        // SINK
        phys = st; nvalid = min(B, v.sink_ntok - st * B);
      } else if (st < n_sink + k_eff) {                         // TOPK[h, i]
        const int32_t e = list[st - n_sink];
        phys = uf_entry_phys(e); nvalid = uf_entry_nvalid(e);
      } else {                                                  // CUR
        const int b = st - n_sink - k_eff;
        phys = v.S + v.cur_slot * v.BPC + b; nvalid = min(B, v.cur_ntok - b * B);
      }
      const __nv_bfloat16* kb = kc + head_base + (int64_t)phys * B * D + lane * EPL;
      const __nv_bfloat16* vb = vc + head_base + (int64_t)phys * B * D + lane * EPL;
      for (int key = 0; key < nvalid; ++key) {
        float part = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) part += qv[e] * __bfloat162float(kb[(int64_t)key * D + e]);
#pragma unroll
        for (int sh = 16; sh > 0; sh >>= 1) part += __shfl_xor_sync(0xffffffffu, part, sh);
        const float s2 = part * sl2;
        const float mn = fmaxf(m, s2);
        const float corr = exp2f(m - mn);                       // exp2f(-inf) = 0 on the first key
        const float p = exp2f(s2 - mn);
        l = l * corr + p;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = acc[e] * corr + p * __bfloat162float(vb[(int64_t)key * D + e]);
        m = mn;
      }
    }
    const float inv = 1.f / l;
#pragma unroll
    for (int e = 0; e < EPL; ++e) o[qoff + e] = __float2bfloat16_rn(acc[e] * inv);
    if (lse && lane == 0) lse[(int64_t)h * v.cur_ntok + i * B + r] = (m + log2f(l)) * 0.6931471805599453f;
  }
}

}  // namespace

cudaError_t uf_launch_attn_generic(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, __nv_bfloat16* o,
                                   float* lse, int64_t tok_stride, int64_t head_stride, float scale,
                                   cudaStream_t s) {
  const int nqb = uf_ceil_div(v.cur_ntok, v.B);
  dim3 grid(nqb, v.H);
#define UF_GEN_CASE(DD)                                                                                     \
  case DD:                                                                                                  \
    uf_attn_generic_kernel<DD><<<grid, kWarps * 32, 0, s>>>(v, q, o, lse, tok_stride, head_stride, c->kc,   \
                                                            c->vc, c->sel_q,                                \
                                                            c->sel_paper ? c->sel_cnt : nullptr, c->kcap,   \
                                                            c->sel_k, scale);                               \
    break;
  switch (v.d) {
    UF_GEN_CASE(32)
    UF_GEN_CASE(64)
    UF_GEN_CASE(128)
    default: return cudaErrorInvalidValue;
  }
#undef UF_GEN_CASE
  c->launches += 1;
  return cudaGetLastError();
}
