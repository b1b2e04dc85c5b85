/* uf.h — C ABI of the B200-native sparse causal chunk attention path of Ultra Flash
 * (arxiv/paper_2606_09150).  Library: paper_2606_09150_b200/libuf.so (built by
 * paper_2606_09150_b200/build.py with nvcc for sm_100a).
 *
 * Citations: `P:NNN` = line NNN of the paper text; `BJ` = BASELINE.json
 * (`north_star`, `configs`); `R-n` = reading n in DESIGN.md §"Readings of the paper".
 *
 * What the path computes, per streaming chunk c of one attention layer (P:86-90, P:136 (iii),
 * P:343; call order "append -> select -> attention" from BJ configs[3]):
 *
 *   uf_kv_append        write the chunk's K,V into a bounded rolling cache, evict the oldest
 *                       chunks under a FIFO window, keep a permanent sink (chunk 0, block 0)
 *   uf_select_blocks    block-mean pool Q and K, score s_ij = qbar_i . kbar_j / sqrt(d) (Eq. 4,
 *                       P:88), keep the top-k cached key blocks per (head, query block)
 *   uf_sparse_attn_fwd  softmax(q k^T / sqrt(d)) v over SINK u TOPK u CUR (the whole current
 *                       chunk), chunk-causal by construction
 *
 * Conventions
 *   - All calls return an int32 status (UF_OK = 0).  uf_last_error() gives a message.
 *   - "device pointer" = CUDA device memory on the ctx's device; "host pointer" = ordinary host
 *     memory.  The caller owns every buffer it passes in; the ctx owns the caches, the pooled-K
 *     table, the selection workspace and the host slot map, all freed by uf_ctx_destroy.
 *   - Device work is enqueued on the caller's stream (`void* stream` = cudaStream_t, NULL = the
 *     legacy default stream) and is asynchronous; host bookkeeping (slot map, candidate set) is
 *     updated synchronously and is valid on return.  Getters that copy device data synchronise
 *     the given stream.
 *   - One ctx = the cache of one (layer, video stream).  A ctx is not thread-safe.
 *   - Q, K, V, O are bf16, logical shape [n_tokens, n_heads, head_dim], element strides
 *     (tok_stride, head_stride, 1); the innermost (head_dim) axis must be contiguous, the base
 *     pointer and both strides*2 bytes must be multiples of 16 bytes.
 *   - Blocks: flat runs of `block` consecutive tokens aligned to the chunk start; the last
 *     block of a chunk may be ragged (R-1, R-3).  Global key-block id g = chunk*BPC + b with
 *     BPC = ceil(chunk_tokens_max / block).
 *   - There is no CPU fallback: every step runs in CUDA kernels for sm_100a.
 */
#ifndef UF_H_
#define UF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define UF_OK               0
#define UF_ERR_INVALID_ARG  1   /* null pointer, bad size/stride/alignment, bad config            */
#define UF_ERR_STATE        2   /* call order: select before append, attn before select, ...      */
#define UF_ERR_CAPACITY     3   /* n_tokens > chunk_tokens_max, window > capacity, buffer too small */
#define UF_ERR_UNSUPPORTED  4   /* shape not covered by any kernel                                 */
#define UF_ERR_CUDA         5   /* a CUDA runtime/driver call failed (message has the CUDA error)  */

#define UF_MAX_CAPACITY_CHUNKS 16

typedef struct uf_ctx uf_ctx;

typedef struct uf_config {
  int32_t n_heads;           /* H  (BJ configs: 1, 12, 40)                                        */
  int32_t head_dim;          /* d  (32, 64 or 128)                                                 */
  int32_t block;             /* B  query block == key block (64 or 128; multiple of 32, <= 128)   */
  int32_t chunk_tokens_max;  /* upper bound on tokens per chunk; BPC = ceil(this / block)         */
  int32_t capacity_chunks;   /* C: resident non-sink chunks INCLUDING the just-appended one (R-16);
                                1..UF_MAX_CAPACITY_CHUNKS.  P:343 "KV cache: 3 temporal windows"  */
  int32_t sink_blocks;       /* S: blocks 0..S-1 of chunk 0 kept forever (BJ configs[0]); 0..4    */
  int32_t k_min;             /* floor on k in percent mode (k_min = 4)                     */
  int32_t device;            /* CUDA ordinal; -1 = host-only ctx: slot-map bookkeeping works,
                                every device step returns UF_ERR_STATE (used by CPU tests)        */
} uf_config;

/* Create a ctx: allocates K cache, V cache ([H][(S + C*BPC)*B][d] bf16, zero-filled), the pooled-K
 * table and the selection workspace on cfg->device.  *out receives the handle. */
int32_t uf_ctx_create(const uf_config* cfg, uf_ctx** out);

/* Free everything the ctx owns.  NULL is accepted. */
int32_t uf_ctx_destroy(uf_ctx* ctx);

/* Start a new video stream: empty cache, no sink, chunk counter back to 0 (R-27).  Host state only:
 * nothing on the device is cleared (every block an append makes addressable is rewritten in full, pad
 * rows as zeros; blocks that are not addressable are never read); `stream` is unused. */
int32_t uf_ctx_reset(uf_ctx* ctx, void* stream);

/* Step a1 — KV append + evict (P:136 (iii) "dynamically selecting a compact cache window",
 * P:343; BJ configs[3] "eviction of the oldest non-sink chunk after each append").
 * The chunk gets id c = number of appends since reset.  With window W = window_chunks (0 -> C,
 * else 1..C) every resident chunk with id <= c - W is evicted, oldest first (FIFO; shrinking W
 * evicts several, growing never resurrects, R-17); the chunk then takes the lowest-numbered free
 * slot.  On c == 0 its first S blocks are also copied to the sink region.  Also produces the
 * block-mean pooled K of the chunk's blocks, used by uf_select_blocks.
 *   k, v        device pointers, bf16 [n_tokens, H, d] with the given element strides
 *   n_tokens    1..chunk_tokens_max
 * If the device work cannot be enqueued (UF_ERR_CUDA) the ctx is left exactly as before the call.
 * With a host-only ctx (device == -1) k, v, stream are ignored and only the slot map advances. */
int32_t uf_kv_append(uf_ctx* ctx, const void* k, const void* v, int32_t n_tokens,
                     int64_t tok_stride, int64_t head_stride, int32_t window_chunks, void* stream);

/* Host query: for the current state, the candidate count |CAND| (blocks of resident chunks older
 * than the newest one, minus the sink ids, R-10/R-15) and the effective budget
 *   k' = min(k, |CAND|),  k = topk_count if topk_count >= 0,
 *                         else max(k_min, floor(topk_percent * |CAND| / 100))   (R-8/R-9).
 * Either output pointer may be NULL. */
int32_t uf_query_topk(const uf_ctx* ctx, int32_t topk_count, int32_t topk_percent,
                      int32_t* n_cand, int32_t* k_eff);

/* Steps a2-a4 — block pooling, scoring (Eq. 4: s_ij^h = qbar_i^h . kbar_j^h / sqrt(d_h), fp64,
 * terms added in index order, no fused multiply-add, R-4) and top-k per (head, query block); equal
 * scores -> the smaller global id wins (BJ); lists ascending by global id.  The selection is kept
 * in the ctx for the following uf_sparse_attn_fwd.  The score is a fixed function of the input bits as long
 * as the block sums are exact in fp64, i.e. the bf16 values of one (block, head, channel) column span fewer
 * than 2^38 between the largest magnitude and the smallest non-zero ulp (8 + 7 + 38 = 53 bits); beyond that
 * the summation order may change the last bit of a pooled mean.
 *   q           device pointer, bf16 [n_tokens, H, d]; n_tokens must equal the last append's
 *   idx_out     device pointer or NULL: int32 [H, ceil(n_tokens/B), k'] global block ids
 *   cnt_out     device pointer or NULL: int32 [H, ceil(n_tokens/B)] (= k' for every row)     */
int32_t uf_select_blocks(uf_ctx* ctx, const void* q, int32_t n_tokens,
                         int64_t tok_stride, int64_t head_stride,
                         int32_t topk_count, int32_t topk_percent,
                         int32_t* idx_out, int32_t* cnt_out, void* stream);

/* Step a5 — block-sparse attention: for every valid query row n of block i and head h
 *   o_n = sum_m softmax_m(q_n . k_m * scale) v_m   over the valid tokens m of
 *   KEPT[h,i] = SINK u TOPK[h,i] u CUR   (BJ north_star; R-13/R-14/R-15).
 * bf16 inputs, fp32 accumulation and softmax, bf16 output (round-to-nearest-even).
 *   q, o        device pointers, bf16 [n_tokens, H, d] (same strides for both)
 *   lse         device pointer or NULL: fp32 [H, n_tokens], natural-log sum-exp of the scaled logits
 *   softmax_scale  0 -> 1/sqrt(d)
 *               o must not overlap q (UF_ERR_INVALID_ARG); disjoint slices of one fused tensor are fine
 * Kernels: B == 128 && d == 128 -> TMA + tcgen05/TMEM kernel.  Other shapes have only the CUDA-core kernel
 * (one warp per query row, orders of magnitude slower): the call returns UF_ERR_UNSUPPORTED unless the caller
 * opted in with uf_set_attn_impl(ctx, 1), which also forces that kernel for B == d == 128 (cross-checks).
 * The tcgen05 path enqueues two
 * launches: the fast kernel (exponentials against the running max of the earlier key blocks) and an
 * exact-max instantiation that redoes the work items in which a row max outgrew that reference by 2^100
 * or more inside one key block (normally none: it returns at once; uf_attn_redone_items reports them).
 * Asynchronous on `stream`; needs softmax_scale >= 0 and finite (else UF_ERR_INVALID_ARG), a preceding
 * uf_select_blocks for the same chunk (else UF_ERR_STATE) and, on the tcgen05 path, 16-byte-aligned q / o
 * with strides that are multiples of 8 elements (TMA; else UF_ERR_INVALID_ARG). */
int32_t uf_sparse_attn_fwd(uf_ctx* ctx, const void* q, void* o, float* lse, int32_t n_tokens,
                           int64_t tok_stride, int64_t head_stride, float softmax_scale,
                           void* stream);

/* ---- Paper-mask mode: the mask exactly as section 2.3.1 / appendix L.1 define it -----
 * P:86  "The 3D token grid (t,h,w) is divided into non-overlapping blocks of (b_t,b_h,b_w) ... a spatial locality
 *        mask M_local confines each block's receptive field to a sliding window of size r x r, and a temporal
 *        causal mask M_causal ensures each temporal chunk attends only to current and preceding chunks"
 * P:88  Eq. 4: M_sparse[i,j] = 1[softmax(s_i,:)_j >= tau_k]  n  M_local  n  M_causal
 * P:815 Eq. 10 (repaired, reading R-34): tau_k = max(k_min, floor(rho * 0.42 * N_blocks))
 * P:343 block (2,8,8), local window 9 x 9, rho = 1.0, k_min = 4.
 * Differences from the default (BASELINE.json) mode: blocks are 3-D tiles of the chunk's token grid (edge tiles
 * ragged, R-29); the candidates of the top-k are ALL blocks in the causal mask, the current chunk's included;
 * the top-k is intersected with the window (R-30/R-32); the query block's own key block is always kept (R-33);
 * there is no sink and no implicitly kept current chunk.
 *
 * Layout: in this mode Q, K, V, O are in TILED order: n_tokens = N_b * block rows, block b = (it*nbh + ih)*nbw + iw
 * (nbt = ceil(F/bt), ...) owns rows [b*block, (b+1)*block), of which the first nvalid(b) hold the tokens of tile
 * (it, ih, iw) that exist, in raster (t, y, x) order inside the tile, and the rest are pad rows (zeros; their O rows
 * are meaningless).  A model keeps its activations in this order for all layers (attention is the only
 * token-mixing op); uf_tile_tokens / uf_untile_tokens convert from / to raster order.  Global id g = chunk*N_b + b. */
typedef struct uf_tiling {
  int32_t frames, grid_h, grid_w;   /* F, Hg, Wg: token grid of one chunk (every chunk the same)               */
  int32_t bt, bh, bw;               /* tile shape; bt*bh*bw must equal uf_config.block (paper: 2, 8, 8)        */
  int32_t window;                   /* r, odd: |dih|, |diw| <= (r-1)/2 in tile coordinates (paper: 9)          */
} uf_tiling;

/* Switch an EMPTY ctx (before the first append, or after uf_ctx_reset) to paper-mask mode.  Needs
 * sink_blocks == 0 and chunk_tokens_max == N_b * block.  Errors: UF_ERR_STATE (cache not empty),
 * UF_ERR_INVALID_ARG (sizes).  From then on uf_kv_append takes tiled chunks of exactly N_b * block rows and
 * uf_select_blocks is replaced by uf_select_blocks_paper. */
int32_t uf_ctx_set_tiling(uf_ctx* ctx, const uf_tiling* tiling);

/* Host query: N_blocks = blocks in the causal mask for the current state (all resident chunks incl. the newest)
 * and the budget k' = min(k, N_blocks), k = topk_count if >= 0 else tau_k(rho_permille / 1000) above.  k' is the
 * size of the top-k BEFORE the window: the blocks a row really keeps are top-k' n M_local plus its own block (the
 * cnt_out of uf_select_blocks_paper), fewer than k' + 1 wherever the window cuts.  The 0.42 of tau_k was read off
 * Table 21's default row as a pre-window fraction; the executed mask is sparser than that column (R-34). */
int32_t uf_query_budget_paper(const uf_ctx* ctx, int32_t topk_count, int32_t rho_permille,
                              int32_t* n_blocks, int32_t* k_eff);

/* Eq. 4 selection for the newest chunk (q in tiled order, as passed to the append): per (head, query tile) the k'
 * best-scoring blocks of the causal mask (fp64 scores as in uf_select_blocks; ties -> lower global id), then only
 * those inside the window, plus the tile's own block.
 *   idx_out   device pointer or NULL: int32 [H, N_b, idx_stride] ascending global ids, padded with -1;
 *             idx_stride >= min(k' + 1, N_blocks) (else UF_ERR_CAPACITY)
 *   cnt_out   device pointer or NULL: int32 [H, N_b] kept blocks per row (1 .. k' + 1)
 * The selection is kept in the ctx for the following uf_sparse_attn_fwd, which then attends exactly these blocks. */
int32_t uf_select_blocks_paper(uf_ctx* ctx, const void* q, int32_t n_tokens,
                               int64_t tok_stride, int64_t head_stride,
                               int32_t topk_count, int32_t rho_permille,
                               int32_t* idx_out, int32_t idx_stride, int32_t* cnt_out, void* stream);

/* Raster [F*Hg*Wg, H, d] -> tiled [N_b*block, H, d] (pad rows written as zeros) and back (pad rows skipped).
 * Device pointers, bf16, element strides as everywhere; src and dst must not overlap.  Asynchronous on `stream`. */
int32_t uf_tile_tokens(uf_ctx* ctx, const void* raster, void* tiled,
                       int64_t raster_tok_stride, int64_t raster_head_stride,
                       int64_t tiled_tok_stride, int64_t tiled_head_stride, void* stream);
int32_t uf_untile_tokens(uf_ctx* ctx, const void* tiled, void* raster,
                         int64_t tiled_tok_stride, int64_t tiled_head_stride,
                         int64_t raster_tok_stride, int64_t raster_head_stride, void* stream);

/* ---- The step in front of the path, fused ------------------------------------------------
 * P:343 "The SR model follows the Wan2.1 architecture ... 12 heads (head dim 128) ... 3D RoPE with axis dims
 * (44,42,42)".  uf_qkv_rope_append takes the raw Q, K, V of the QKV projection and, in ONE pass over them, does what
 * otherwise takes an elementwise kernel, uf_kv_append and the pooling pass of uf_select_blocks (readings R-37..R-40):
 *   QK-norm  y = x / sqrt(mean over the token's H*d channels of x^2 + eps) * g   (q with gq, k with gk; v untouched)
 *   RoPE     channel pairs (2i, 2i+1) of every head are complex numbers multiplied by cos + i sin of
 *            pos * theta^(-2 i_a / D_a): the first dim_t/2 pairs follow the token's frame t0 + t, the next dim_h/2 its
 *            row y, the last dim_w/2 its column x; the cos / sin values come from the caller's tables (model state)
 *   round    to bf16 (nearest even).  Everything before it is IEEE fp32, each operation rounded once, no fused
 *            multiply-add, in the stated order (the sum of squares and the reciprocal square root run in fp64 and are
 *            rounded to fp32 once), so cache bytes and block indices are a fixed function of the input bits; against
 *            the fp64 definition (one rounding) the result is equal or adjacent in bf16 (within one ulp)
 *   write    post-RoPE Q -> q_out; post-RoPE K and V -> the cache slot, exactly as uf_kv_append (same eviction policy,
 *            sink copy, zero pad rows); block-mean pooled K and pooled Q -> the ctx.
 * A following uf_select_blocks / uf_select_blocks_paper called with q == q_out (same strides) skips its pooling
 * pass: it is recognised by ADDRESS AND STRIDES ONLY, so the buffer must still hold, bit for bit, what this call
 * wrote.  A caller that rewrites q_out (or reuses its memory for another Q) between the two calls must switch the
 * shortcut off with uf_set_pooled_q_reuse(ctx, 0); otherwise the selection is made for the Q this call wrote, not for
 * the q argument, and no error is raised.
 * Aliasing: q_out may be q_in itself (same pointer and strides: in place); any other overlap of q_out with q_in,
 * k_in or v_in is refused (UF_ERR_INVALID_ARG).  Disjoint slices of one fused tensor are fine.  Token positions: raster order (t, y, x) over a grid_h x grid_w grid (token n: t = t0 + n / (gh*gw), ...); on a
 * tiled ctx the tiling's grid and order are used and grid_h / grid_w are ignored.  head_dim must be 128.
 * Errors as uf_kv_append, plus UF_ERR_CAPACITY when a position exceeds max_pos. */
typedef struct uf_rope_spec {
  const float* cos_tab;       /* device, fp32 [max_pos][head_dim/2]: column i = cos(row * freq_i)             */
  const float* sin_tab;       /* device, fp32 [max_pos][head_dim/2]                                            */
  const float* gq;            /* device, fp32 [n_heads*head_dim]: RMSNorm weight of q                          */
  const float* gk;            /* device, fp32 [n_heads*head_dim]: RMSNorm weight of k                          */
  double eps;                 /* 1e-6                                                                           */
  int32_t max_pos;            /* rows of the tables                                                             */
  int32_t t0;                 /* temporal position of the chunk's first latent frame (chunk c: c * F)          */
  int32_t grid_h, grid_w;     /* token grid (raster mode)                                                       */
  int32_t dim_t, dim_h, dim_w;/* axis dims, even, sum = head_dim (paper: 44, 42, 42)                            */
} uf_rope_spec;

int32_t uf_qkv_rope_append(uf_ctx* ctx, const void* q_in, const void* k_in, const void* v_in, void* q_out,
                           int32_t n_tokens, int64_t in_tok_stride, int64_t in_head_stride,
                           int64_t out_tok_stride, int64_t out_head_stride,
                           const uf_rope_spec* rope, int32_t window_chunks, void* stream);

/* on != 0 (default): a select called with the q_out pointer and strides of the chunk's uf_qkv_rope_append reuses the
 * pooled Q that call produced.  on == 0: every select pools the q it is given (one more small kernel per call). */
int32_t uf_set_pooled_q_reuse(uf_ctx* ctx, int32_t on);

/* ---- SR cache window policy --------------------------------------------------------------
 * The paper states the idea three times and gives no rule: P:136 (iii) "dynamically selecting a compact cache window,
 * trading minimal quality for significant memory and compute savings", "SR cache window: dynamically selected
 * based on content complexity", "Select compact SR KV window based on chunk position and memory budget".
 * Reading R-36: one small host function maps a stated policy to the `window_chunks` argument of the
 * NEXT uf_kv_append; the mechanism (FIFO, shrinking evicts several, growing never resurrects) is R-17's.
 *   UF_WIN_FIXED     W = C.
 *   UF_WIN_POSITION  W = C for chunks 0 .. warm_chunks-1, compact_window afterwards ("chunk position").
 *   UF_WIN_MEMORY    W = floor(budget_bytes / bytes of one cache slot), slot = K + V = 2 * H * BPC * B * d * 2 bytes
 *                    ("memory budget"); clamped to 1 .. C.
 *   UF_WIN_CONTENT   ("content complexity") uses an exact integer statistic of the LAST selection: how many of the kept
 *                    top-k blocks, over all heads and query blocks, lie in each listed chunk (uf_get_select_usage).
 *                    T = min(C, resident + 1) chunks would be resident after the next append under plain FIFO (its
 *                    victim, if the cache is full, goes anyway).  Then, oldest survivor first: while that chunk holds
 *                    fewer than min_share_permille of the kept blocks and T > compact_window, it is evicted too
 *                    (T -= 1).  W = T.  Content whose top-k picks concentrate on recent chunks thus runs with a short
 *                    window; the window grows again (by one chunk per append) when old chunks are being used.
 * All results are clamped to 1 .. C.  UF_WIN_CONTENT synchronises `stream` (it reads 128 bytes of counters);
 * a caller evaluates it once per chunk (on one layer) and applies the window to every layer.  The rule itself has
 * no counterpart in the paper to check against: parity unpinned for the RULE; the statistic and the integer
 * arithmetic are compared bit-exactly with oracle/uf_window_policy.py. */
#define UF_WIN_FIXED     0
#define UF_WIN_POSITION  1
#define UF_WIN_MEMORY    2
#define UF_WIN_CONTENT   3

typedef struct uf_window_policy {
  int32_t kind;                /* UF_WIN_*                                                             */
  int32_t warm_chunks;         /* POSITION                                                             */
  int32_t compact_window;      /* POSITION: W after the warm phase; CONTENT: smallest resident count   */
  int32_t min_share_permille;  /* CONTENT: 0 .. 1000                                                   */
  int64_t budget_bytes;        /* MEMORY: cap on resident non-sink K + V cache bytes                   */
} uf_window_policy;

/* window_chunks (host pointer) receives the W to pass to the next uf_kv_append. */
int32_t uf_next_window(uf_ctx* ctx, const uf_window_policy* policy, int32_t* window_chunks, void* stream);

/* Kept top-k blocks of the last selection per listed chunk (ascending chunk id; the candidates' chunks: resident
 * prior chunks, in paper-mask mode also the newest).  Host outputs: kept_per_chunk[n], chunk_ids[n] (either may be
 * NULL), *n_chunks = n <= capacity.  Synchronises `stream`.  UF_ERR_STATE without a valid selection. */
int32_t uf_get_select_usage(uf_ctx* ctx, int64_t* kept_per_chunk, int32_t* chunk_ids, int32_t* n_chunks,
                            void* stream);

/* impl: 0 = tcgen05 kernel only (default; shapes it does not cover -> UF_ERR_UNSUPPORTED),
 *       1 = the generic CUDA-core attention kernel (any supported shape; slow),
 *       2 = the CTA-pair tcgen05 kernel (cta_group::2 MMAs over two CTAs, one query tile per CTA, each CTA loads half of
 *           every K / V tile, triple-buffered S, two softmax warp groups per CTA taking the key blocks in turn; same
 *           shapes and results as 0 within the tolerance; measured 3-5 % slower on B200, kept selectable: DESIGN.md 5.1). */
int32_t uf_set_attn_impl(uf_ctx* ctx, int32_t impl);

/* Observability (host outputs).
 * uf_get_slot_map: slot_chunk[C] = chunk id resident in each slot or -1; n_resident; newest chunk
 * id (-1 before the first append).  Any pointer may be NULL. */
int32_t uf_get_slot_map(const uf_ctx* ctx, int32_t* slot_chunk, int32_t* n_resident,
                        int32_t* newest_chunk);

/* uf_get_cache_block: copy the cached K and V rows of one key block and one head to host memory.
 * global_block: g = chunk*BPC + b of a resident chunk, or -(s+1) for sink block s.
 * k_out, v_out: host pointers (or NULL), bf16 [B, d]; rows past the block's valid count are the
 * cache's zero padding.  Synchronises `stream`. */
int32_t uf_get_cache_block(uf_ctx* ctx, int32_t global_block, int32_t head,
                           void* k_out, void* v_out, void* stream);

/* uf_get_pooled_k: copy the block-mean pooled K (fp64 [d]) of one resident key block and head to
 * host memory (same addressing as uf_get_cache_block).  Synchronises `stream`. */
int32_t uf_get_pooled_k(uf_ctx* ctx, int32_t global_block, int32_t head, double* out, void* stream);

/* uf_attn_redone_items: how many work items (head, query-block pair) of the LAST uf_sparse_attn_fwd call
 * were redone by the exact-max ("safe") instantiation of the tcgen05 attention kernel because a row
 * max outgrew the running reference by 2^100 or more within one key block.  Writes the
 * count to host memory `*n_items` (0 for the generic kernel).  Synchronises `stream`. */
int32_t uf_attn_redone_items(uf_ctx* ctx, int32_t* n_items, void* stream);

/* Bytes of device memory the ctx owns. */
int64_t uf_ctx_device_bytes(const uf_ctx* ctx);

/* Number of kernels the ctx has launched since creation (bench.py's gpu_launches). */
int64_t uf_ctx_launch_count(const uf_ctx* ctx);

/* Message of the last failing call on this ctx (ctx-owned string; "" if none).  With ctx == NULL:
 * message of the last failing uf_ctx_create on this thread. */
const char* uf_last_error(const uf_ctx* ctx);

/* Library version string, e.g. "uf-b200 0.1 (sm_100a)". */
const char* uf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* UF_H_ */
