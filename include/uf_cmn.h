/* uf_cmn.h — C ABI of the causal memory network streaming step of Ultra Flash:
 * the streaming latent upsampler and the HR decoder of paper section 2.2, Eq. 2,
 * Algorithm 2, configurations P:345-347: VARIANT A's function (the memory of a block is its INPUT one
 * frame earlier, line 7 at P:482), evaluated as a stream with the state variant B keeps (one memory per block in the
 * handle).  It is NOT variant B as printed: lines 31-32 store the block OUTPUT, a recurrence over frames
 * that is a different function from the second frame on (reading R-41; oracle/uf_causal_mem.py
 * CausalMemStream(memory="output") is that literal form, and tests/test_causal_mem_pins.py pins the difference).
 * Weights trained against the literal variant B are not served by this call.  Same library as uf.h
 * (paper_2606_09150_b200/libuf.so); status codes and conventions are those of uf.h.
 *
 * What one uf_cmn_step computes, for the next n_frames input frames z of a video stream:
 *
 *   h = Conv3x3_in(z)
 *   per stage s:  N_b CausalMemBlocks (Eq. 2)
 *                   h <- relu( Conv3(Conv2(relu(Conv1([h ; m])))) + W_skip h ),
 *                   m = the block's input one frame earlier (zeros before the first frame; the last frame's
 *                   input is kept in the handle for the next call: R-41 in DESIGN.md)
 *                 h <- PixelShuffle_r(Conv3x3_up(h));  if s_s > 1: h <- channel-to-time(Conv1x1_texp(h));
 *                 h <- Conv1x1_ch(h)
 *   out = Conv3x3_out(h)
 *
 * Arithmetic (R-46): bf16 activations and weights, fp32 accumulation on the tcgen05 tensor cores (every
 * convolution is an implicit GEMM: 128 output pixels x C_out x (taps * C_in)), fp32 bias, ReLU, ONE rounding
 * to bf16 per layer output; Conv3 and W_skip of a block accumulate into the same sum.  Zero padding,
 * cross-correlation (R-42); PixelShuffle and channel-to-time index conventions R-44.
 *
 * Layout: activations are bf16 [frames, rows, columns, channels] (channels innermost), dense.
 * Supported shapes: every entry of stage_channels a multiple of 64 and <= 256; in_ch, out_ch <= 64 with in_ch
 * a multiple of 8; spatial factors 1..3; temporal factors 1..4; C * r^2 and C * s multiples of 64.  Anything
 * else: UF_ERR_UNSUPPORTED from uf_cmn_create.  There is no CPU fallback.
 */
#ifndef UF_CMN_H_
#define UF_CMN_H_

#include <stdint.h>

#include "uf.h"

#ifdef __cplusplus
extern "C" {
#endif

#define UF_CMN_MAX_STAGES 4

typedef struct uf_cmn uf_cmn;

typedef struct uf_cmn_config {
  int32_t in_ch, out_ch;                             /* 16 / 16; 16 / 3                         */
  int32_t n_stages;                                  /* 1 .. UF_CMN_MAX_STAGES                                 */
  int32_t stage_channels[UF_CMN_MAX_STAGES + 1];     /* width of stage s; entry n_stages = width after the last
                                                        channel transition, 0 = same as the last stage (R-45)  */
  int32_t n_blocks;                                  /* N_b CausalMemBlocks per stage (3)               */
  int32_t spatial_factors[UF_CMN_MAX_STAGES];        /* r_s                                                     */
  int32_t temporal_factors[UF_CMN_MAX_STAGES];       /* s_s                                                     */
  int32_t height, width;                             /* input grid (rows, columns)                              */
  int32_t frames_max;                                /* most input frames one uf_cmn_step may take              */
  int32_t device;                                    /* CUDA ordinal                                            */
} uf_cmn_config;

/* Create a network handle: allocates activation buffers, the per-block memories (zeroed) and the packed weight
 * matrices on `device`.  *out is set on UF_OK.  With out == NULL or cfg == NULL: UF_ERR_INVALID_ARG.             */
int32_t uf_cmn_create(const uf_cmn_config* cfg, uf_cmn** out);
int32_t uf_cmn_destroy(uf_cmn* n);

/* Parameters.  Names: "in", "s<S>.b<B>.c1|c2|c3|skip", "s<S>.up", "s<S>.texp" (only when s_s > 1), "s<S>.ch",
 * "out" (Alg. 2's Conv^in, Conv^(1..3), W_skip, Conv^up, Conv^texp, Conv^ch, Conv^out).  Shapes are the usual
 * [C_out, C_in, 3, 3] (3x3) or [C_out, C_in, 1, 1] (1x1); "c1" has C_in = 2C: first C = h, next C = memory.
 * uf_cmn_n_params / uf_cmn_param_info enumerate them in network order.  uf_cmn_set_param takes HOST pointers:
 * w = bf16 [C_out, C_in, kh, kw] contiguous, bias = fp32 [C_out] or NULL (must be NULL for "skip", R-43; NULL
 * elsewhere means zero).  It repacks into the kernel's GEMM layout and copies to the device synchronously.
 * Unknown name: UF_ERR_INVALID_ARG.                                                                              */
int32_t uf_cmn_n_params(const uf_cmn* n);
int32_t uf_cmn_param_info(const uf_cmn* n, int32_t index, char* name, int32_t name_cap, int32_t shape[4],
                          int32_t* has_bias);
int32_t uf_cmn_set_param(uf_cmn* n, const char* name, const void* w_host, const float* bias_host);

/* Start a new video stream: every block memory becomes zero (Alg. 2 line 23).  Host bookkeeping only (the next step
 * reads an all-zero frame kept in every memory buffer); `stream` is unused.                                          */
int32_t uf_cmn_reset(uf_cmn* n, void* stream);

/* One streaming step (Alg. 2 lines 24-41 for n_frames consecutive frames).
 *   z    device, bf16 [n_frames, height, width, in_ch], 16-byte aligned
 *   out  device, bf16 [n_frames * prod(s_s), height * prod(r_s), width * prod(r_s), out_ch]
 * 1 <= n_frames <= frames_max (else UF_ERR_CAPACITY); every parameter must have been set (else UF_ERR_STATE).
 * All kernels are enqueued on `stream`; the memories are updated by the same stream, so steps of one handle
 * must be issued in stream order.                                                                                 */
int32_t uf_cmn_step(uf_cmn* n, const void* z, int32_t n_frames, void* out, void* stream);

/* Observability: copy the memory of block `block` of stage `stage` (the block's input at the last frame seen)
 * to HOST memory, bf16 [rows_s, cols_s, C_s]; synchronises `stream`.  shape_out (nullable) receives
 * {rows_s, cols_s, C_s}.                                                                                          */
int32_t uf_cmn_get_memory(uf_cmn* n, int32_t stage, int32_t block, void* out_host, int32_t shape_out[3],
                          void* stream);

/* Observability: the output of layer `layer` (index as in uf_cmn_layer_info; PixelShuffle / channel-to-time already
 * applied) for the frames of the LAST uf_cmn_step, to HOST memory, bf16 [frames_l, rows_l, cols_l, C_l]; shape_out
 * (nullable) receives that shape.  Call it with out_host sized for frames_max * prod(s_s) frames, or query the shape
 * of a smaller step first by its layer info.  The last layer ("out") writes the caller's tensor and has no buffer:
 * UF_ERR_INVALID_ARG.  Before any step: UF_ERR_STATE.  Synchronises `stream`.                                       */
int32_t uf_cmn_get_activation(uf_cmn* n, int32_t layer, void* out_host, int32_t shape_out[4], void* stream);

/* 2 * multiply-adds of all convolutions for n_frames input frames, real channel counts (no padding).             */
int64_t uf_cmn_flops(const uf_cmn* n, int32_t n_frames);
int64_t uf_cmn_device_bytes(const uf_cmn* n);
/* kernels launched by this handle so far (bench.py's gpu_launches)                                               */
int64_t uf_cmn_launches(const uf_cmn* n);
/* number of layers (= kernel launches of one step); per layer: its name ("in", "s0.b0.c1", "s0.b0.c2",
 * "s0.b0.c3+skip", ..., "s0.up", "s0.texp", "s0.ch", ..., "out"), 2 * multiply-adds per INPUT frame, the GEMM's N and K
 * as the kernel runs it (padded), and out_shape (nullable) = {frames per input frame, rows, cols, channels} of its
 * output tensor                                                                                                    */
int32_t uf_cmn_n_layers(const uf_cmn* n);
int32_t uf_cmn_layer_info(const uf_cmn* n, int32_t index, char* name, int32_t name_cap, int64_t* flops_per_frame,
                          int32_t* gemm_n, int32_t* gemm_k, int32_t out_shape[4]);
const char* uf_cmn_last_error(const uf_cmn* n);

#ifdef __cplusplus
}
#endif
#endif  /* UF_CMN_H_ */
