/* uf_static.h — block selection for callers that must not allocate device memory.
 *
 * Who this is for.  Everything in uf.h goes through a uf_ctx, and uf_ctx_create cudaMallocs the caches and the
 * selection workspace.  Some hosts of this library cannot do that:
 *   - an inference-runtime plug-in whose per-step hook runs under a "no allocation here" contract (the runtime hands
 *     the plug-in its inputs and outputs and nothing else);
 *   - a process in which another framework's caching allocator has already claimed the GPU's memory, so that a
 *     cudaMalloc from this library would fail or fight that allocator for what is left;
 *   - a latency-critical loop that cannot take the device-wide synchronisation a cudaMalloc / cudaFree implies.
 * For them there is ONE call, uf_select_blocks_static: steps a2-a4 of the path (block-mean pooling, Eq. 4 scores,
 * exact top-k; P:88-90 of the paper text) on the caller's Q and K, with the pooled tables — the only intermediate
 * the selection needs — kept in a fixed array that is part of the library image instead of in memory obtained at
 * run time.  It calls no cudaMalloc / cudaFree and no library routine that allocates.
 *
 * The array.  UF_STATIC_SCRATCH_BYTES (16 MiB) of `static __device__` storage in uf_select_static.cu.  Every GPU on
 * which this library's code is loaded carries it until the process exits, whether or not the call is ever used.
 * Problems whose pooled tables do not fit are refused (UF_ERR_CAPACITY), never spilled anywhere else:
 *   needed bytes = roundup256(8 * H * d * nqb) + 8 * H * d * nkb,  nqb = ceil(n_q_tokens / B), nkb = ceil(n_k_tokens / B)
 *   and nkb <= UF_STATIC_MAX_KEY_BLOCKS (the keys of one query block are ranked in shared memory).
 * BASELINE.json configs[1] (H 12, d 128, B 128, 255 query blocks against two cached chunks = 510 key blocks) needs
 * 9.4 MB and fits; configs[2] (2K) does not.
 *
 * Sharing.  All calls, from every thread and on every stream, use the same array on a given GPU, and it is never
 * cleared between calls: it holds whatever the previous call left.  That is harmless for one call at a time, because
 * each call writes every pooled value before it reads it (nothing in the array has to start at zero, so nothing is
 * cleared).  It is NOT harmless for two calls whose kernels can run at the same time on one GPU — two streams, or two
 * host threads — those race on the array and both results are garbage.  Order such calls yourself (one stream, or an
 * event between them).  Calls on different GPUs do not interact.
 *
 * First call on a GPU.  The library needs the array's device address; it asks the CUDA runtime for it
 * (cudaGetSymbolAddress, with that GPU current) the first time the call runs on each GPU and remembers the answer.
 * That first call also makes the driver load this file's kernels.  Make it early — during start-up, and before any
 * stream capture is begun — so that later calls only enqueue kernels.
 */
#ifndef UF_STATIC_H_
#define UF_STATIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define UF_STATIC_SCRATCH_BYTES   (16 * 1024 * 1024)
#define UF_STATIC_MAX_KEY_BLOCKS  4096

/* Select, for every head h and every query block i, the `topk_count` key blocks with the largest
 *   s_ij = qbar_i . kbar_j / sqrt(d)          (Eq. 4; qbar, kbar = means over the valid rows of a block)
 * among ALL nkb key blocks of k; equal scores go to the smaller block index; each output row is ascending.
 * Arithmetic is the one uf_select_blocks uses (exact fp64 block sums, one division for the mean, products and sums
 * rounded separately in channel order, one division by sqrt(d)), so for the same Q and the same candidate blocks the
 * two return the same indices bit for bit.  There is no cache, no sink and no window here: the caller passes the
 * keys to choose from, and block j is rows [j*B, min((j+1)*B, n_k_tokens)) of k.
 *   device        CUDA ordinal the pointers live on; made current by the call
 *   q, k          device pointers, bf16, logical [n_tokens, n_heads, head_dim] with element strides
 *                 (tok_stride, head_stride, 1); 16-byte aligned, strides multiples of 8 and >= head_dim; finite values
 *   head_dim      32, 64 or 128;  block: 32, 64, 96 or 128
 *   topk_count    >= 1; k' = min(topk_count, nkb) entries are written per row
 *   idx_out       device pointer, int32 [n_heads][nqb][k'], block indices into k
 *   stream        cudaStream_t (NULL = legacy default stream); the two kernels are enqueued on it, asynchronously
 * Returns UF_OK or an error code of uf.h: UF_ERR_INVALID_ARG (pointers, strides, sizes), UF_ERR_CAPACITY (does not
 * fit the array / too many key blocks — checked before anything touches the GPU), UF_ERR_CUDA.  The caller owns
 * q, k and idx_out; nothing else outlives the call except the pooled tables in the shared array. */
int32_t uf_select_blocks_static(int32_t device,
                                const void* q, int32_t n_q_tokens, int64_t q_tok_stride, int64_t q_head_stride,
                                const void* k, int32_t n_k_tokens, int64_t k_tok_stride, int64_t k_head_stride,
                                int32_t n_heads, int32_t head_dim, int32_t block, int32_t topk_count,
                                int32_t* idx_out, void* stream);

/* Message of the last failing uf_select_blocks_static on the calling thread ("" if none).  The string lives in
 * thread-local storage of the library (no heap). */
const char* uf_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* UF_STATIC_H_ */
