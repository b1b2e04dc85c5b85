// uf_internal.h — shared declarations of the CUDA path (not part of the ABI; see include/uf.h).
// Notation follows DESIGN.md: H heads, d head_dim, B block, BPC blocks per chunk slot, C capacity,
// S sink blocks, P = S + C*BPC physical key blocks per head, g = chunk*BPC + b global block id.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda.h>
#include <stdint.h>

#include <string>

#include "uf.h"

#define UF_MAXC UF_MAX_CAPACITY_CHUNKS

// Physical layout of the K cache and of the V cache (ctx-owned):
//   [head h][physical token row = phys*B + r][d] bf16,  phys in [0, P):
//   phys 0..S-1 = sink region, phys S + slot*BPC + b = block b of the chunk resident in `slot`.
// Every key block is one contiguous B x d tile, so a single tiled TMA load at token coordinate
// phys*B fetches it.  Rows past a block's valid count are zero.

// A key-block reference handed to the attention kernels, packed in one int32:
//   bits  0..19  phys     physical block index
//   bits 20..27  nvalid-1 valid key rows in the block (1..B)
//   bits 28..29  mask     which of the CTA's two query tiles attend it (sm100 kernel only)
__host__ __device__ inline int32_t uf_entry_pack(int phys, int nvalid, int mask) {
  return (int32_t)((uint32_t)phys | ((uint32_t)(nvalid - 1) << 20) | ((uint32_t)mask << 28));
}
__host__ __device__ inline int uf_entry_phys(int32_t e)   { return (int)((uint32_t)e & 0xFFFFFu); }
__host__ __device__ inline int uf_entry_nvalid(int32_t e) { return (int)(((uint32_t)e >> 20) & 0xFFu) + 1; }
__host__ __device__ inline int uf_entry_mask(int32_t e)   { return (int)(((uint32_t)e >> 28) & 0x3u); }

// Paper-mask mode (R-29/R-30): every chunk is a (nbt x nbh x nbw) grid of (bt, bh, bw) tiles over an
// (F, Hg, Wg) token grid; block b = (it*nbh + ih)*nbw + iw holds the tokens of its tile that exist, in
// raster order, at rows [0, nvalid) of a B-row block (the caller's Q/K/V/O are in this tiled, padded layout).
struct UfTiling {
  int enabled;                    // 0: flat blocks of B consecutive tokens (BJ)
  int F, Hg, Wg, bt, bh, bw;
  int nbt, nbh, nbw;
  int half;                       // (r - 1) / 2: M_local keeps |dih| <= half and |diw| <= half
};
__host__ __device__ inline void uf_tile_coords(const UfTiling& t, int b, int* it, int* ih, int* iw) {
  *it = b / (t.nbh * t.nbw);
  const int rem = b - *it * (t.nbh * t.nbw);
  *ih = rem / t.nbw;
  *iw = rem - *ih * t.nbw;
}
__host__ __device__ inline int uf_tile_nvalid(const UfTiling& t, int b) {
  int it, ih, iw;
  uf_tile_coords(t, b, &it, &ih, &iw);
  const int vt = t.F - it * t.bt < t.bt ? t.F - it * t.bt : t.bt;
  const int vh = t.Hg - ih * t.bh < t.bh ? t.Hg - ih * t.bh : t.bh;
  const int vw = t.Wg - iw * t.bw < t.bw ? t.Wg - iw * t.bw : t.bw;
  return vt * vh * vw;
}
__host__ __device__ inline bool uf_tile_local(const UfTiling& t, int bi, int bj) {
  int ti, hi, wi, tj, hj, wj;
  uf_tile_coords(t, bi, &ti, &hi, &wi);
  uf_tile_coords(t, bj, &tj, &hj, &wj);
  const int dh = hi > hj ? hi - hj : hj - hi, dw = wi > wj ? wi - wj : wj - wi;
  return dh <= t.half && dw <= t.half;
}

// Snapshot of the cache state for one step, passed by value to kernels.
struct UfView {
  UfTiling til;
  int H, d, B, BPC, S, P;
  int n_prior;                    // resident chunks older than the current one, ascending id
  int prior_chunk[UF_MAXC];       // chunk id
  int prior_slot[UF_MAXC];        // slot it lives in
  int prior_ntok[UF_MAXC];        // its token count
  int prior_first_b[UF_MAXC];     // first block that is a candidate (sink ids are skipped, R-15)
  int cand_prefix[UF_MAXC + 1];   // candidates contributed by priors [0, i)
  int n_cand;                     // |CAND|
  int cur_chunk, cur_slot, cur_ntok;
  int n_sink_blocks;              // sink blocks attended this step (0 for chunk 0: inside CUR)
  int sink_ntok;                  // valid tokens in the sink region
};

__host__ __device__ inline int uf_ceil_div(int a, int b) { return (a + b - 1) / b; }

// candidate j (ascending global id) -> global id, physical block, valid rows
__host__ __device__ inline void uf_cand_lookup(const UfView& v, int j, int* g, int* phys, int* nvalid) {
  int i = 0;
  while (i + 1 < v.n_prior && j >= v.cand_prefix[i + 1]) ++i;
  int b = v.prior_first_b[i] + (j - v.cand_prefix[i]);
  *g = v.prior_chunk[i] * v.BPC + b;
  *phys = v.S + v.prior_slot[i] * v.BPC + b;
  int rem = v.prior_ntok[i] - b * v.B;
  *nvalid = v.til.enabled ? uf_tile_nvalid(v.til, b) : (rem < v.B ? rem : v.B);
}

// index (into the view's prior list, ascending chunk id) of the chunk candidate j belongs to
__host__ __device__ inline int uf_cand_prior(const UfView& v, int j) {
  int i = 0;
  while (i + 1 < v.n_prior && j >= v.cand_prefix[i + 1]) ++i;
  return i;
}

// valid rows of block b of the current chunk
__host__ __device__ inline int uf_cur_nvalid(const UfView& v, int b) {
  if (v.til.enabled) return uf_tile_nvalid(v.til, b);
  const int rem = v.cur_ntok - b * v.B;
  return rem < v.B ? rem : v.B;
}

struct uf_ctx {
  uf_config cfg;
  int BPC = 0, P = 0;
  bool host_only = false;
  // device buffers
  __nv_bfloat16* kc = nullptr;    // K cache [H][P*B][d]
  __nv_bfloat16* vc = nullptr;    // V cache [H][P*B][d]
  double* kpool = nullptr;        // block-mean pooled K, [H][d][P] (transposed for coalesced scoring)
  double* qbar = nullptr;         // block-mean pooled Q of the current chunk, [H][BPC][d]
  int32_t* sel_q = nullptr;       // per (h, q-block): k' packed entries, ascending global id; [H][BPC][kcap]
  int32_t* sel_rank = nullptr;    // candidate index of every sel_q entry (merge key); [H][BPC][kcap]
  int32_t* sel_pair = nullptr;    // per (h, q-block pair): merged union list with tile masks; [H][NP][2*kcap]
  int32_t* pair_cnt = nullptr;    // [H][NP]
  unsigned long long* usage = nullptr;   // [2][UF_MAXC]: kept blocks per listed chunk in the last selection (NEXT-3);
                                         // buffer usage_seq & 1 is current, the other one is zeroed for the next call
  int usage_seq = 0;
  int usage_chunk[UF_MAXC];       // chunk ids the current usage buffer refers to (host)
  int usage_n = 0;
  int qbar_chunk = -1;            // chunk whose pooled Q is already in qbar (written by uf_qkv_rope_append), or -1
  const void* qbar_ptr = nullptr; // ... for this post-RoPE Q buffer and these strides
  int64_t qbar_ts = 0, qbar_hs = 0;
  bool skip_pool_q = false;       // set per select call: qbar is valid for the q passed in
  bool reuse_pooled_q = true;     // uf_set_pooled_q_reuse: a select may skip its pooling pass (see uf.h)
  int32_t* sel_cnt = nullptr;     // [H][BPC]: entries of every sel_q row (paper-mask mode: rows differ in length)
  UfTiling til = {};              // paper-mask mode when til.enabled
  bool sel_paper = false;         // the stored selection came from uf_select_blocks_paper
  int32_t* panic_item = nullptr;  // [H][NP]: == attn_seq when the safe attention kernel must redo the item
  int32_t* panic_last = nullptr;  // [1]: == attn_seq when the last fast launch flagged anything
  int32_t attn_seq = 0;           // sm100 attention launch sequence number
  bool last_attn_sm100 = false;   // the last uf_sparse_attn_fwd ran the sm100 kernels
  int kcap = 0;                   // (C-1)*BPC
  int64_t dev_bytes = 0;
  // host state
  int slot_chunk[UF_MAXC];
  int slot_ntok[UF_MAXC];
  int next_chunk = 0;
  int sink_ntok = 0;
  bool sel_valid = false;
  int sel_k = 0, sel_ntok = 0;
  int attn_impl = 0;
  int64_t launches = 0;
  int sm_count = 0;
  CUtensorMap tm_k, tm_v;         // K / V cache maps for the sm100 kernel (valid when B == d == 128)
  CUtensorMap tm_k_half;          // K cache map with 64-row boxes (the CTA-pair kernel loads half a K tile per CTA)
  bool tm_ok = false;
  // Q / O tensor maps of recent callers, keyed by (pointer, rows, strides): a model calls with the same few
  // buffers for every layer and chunk, so cuTensorMapEncodeTiled runs once per buffer, not twice per call
  struct TmEntry { const void* ptr; int64_t tok_stride, head_stride; int rows; CUtensorMap map; };
  static constexpr int kTmCache = 8;
  TmEntry tm_cache[kTmCache];
  int tm_cache_n = 0, tm_cache_next = 0;
  size_t score_smem_attr[4][3][4] = {};   // dynamic-smem limit already set on uf_score_topk_kernel<d, QG>
  size_t fused_smem_attr[4] = {};         // ... on the four uf_fused_append_kernel instantiations (this ctx's device)
  std::string err;
};

// --- kernels (each launcher returns cudaGetLastError()) -------------------------------------------
cudaError_t uf_launch_append(uf_ctx* c, const UfView& v, const __nv_bfloat16* k, const __nv_bfloat16* vv,
                             int64_t tok_stride, int64_t head_stride, cudaStream_t s);
// paper: Eq. 4 mode (candidates include the current chunk, top-k then M_local, own block always kept;
// idx_out rows are out_stride entries long, padded with -1)
cudaError_t uf_launch_select(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, int64_t tok_stride,
                             int64_t head_stride, int k_eff, int32_t* idx_out, int32_t* cnt_out,
                             bool paper, int out_stride, cudaStream_t s);
cudaError_t uf_launch_fused_append(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, const __nv_bfloat16* k,
                                   const __nv_bfloat16* vv, __nv_bfloat16* q_out, int64_t in_ts, int64_t in_hs,
                                   int64_t out_ts, int64_t out_hs, const uf_rope_spec* rs, cudaStream_t s);
// raster [F*Hg*Wg, H, d] <-> tiled, padded [NB*B, H, d] (pad rows zero)
cudaError_t uf_launch_tile(uf_ctx* c, const __nv_bfloat16* src, __nv_bfloat16* dst, int64_t src_tok_stride,
                           int64_t src_head_stride, int64_t dst_tok_stride, int64_t dst_head_stride, bool untile,
                           cudaStream_t s);
cudaError_t uf_launch_attn_generic(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, __nv_bfloat16* o,
                                   float* lse, int64_t tok_stride, int64_t head_stride, float scale,
                                   cudaStream_t s);
// returns UF_* status (tensor-map encoding can fail); message in c->err
int uf_launch_attn_sm100(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, __nv_bfloat16* o, float* lse,
                         int64_t tok_stride, int64_t head_stride, float scale, cudaStream_t s);
int uf_sm100_make_cache_maps(uf_ctx* c);
