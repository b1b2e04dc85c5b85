// uf_cmn.cu — the causal memory network streaming step (include/uf_cmn.h; paper section 2.2, Eq. 2 P:65,
// Alg. 2: variant A's function — memory = block input one frame earlier, R-41 — streamed with per-block state): every convolution of the network as an implicit GEMM on the tcgen05 tensor cores.
//
// One kernel serves all layers.  GEMM view of a layer: M = output pixels (tiles of 128 = 8 rows x 16 columns of one
// frame), N = output channels (<= 256 per tile), K = sum over the layer's sources of taps x channels:
//   Conv1 of a block   : sources (h, 3x3) and (memory = h one frame earlier, 3x3)      [h ; m] of Eq. 2
//   Conv3 + W_skip     : sources (a2, 3x3) and (h, 1x1), one accumulator, one rounding
//   everything else    : one source, 3x3 or 1x1
// A operand: activations are bf16 [frame][row][column][channel]; a 4-D tiled TMA load of a 64-channel x 16-column
//   x R-row box lands in shared memory as R*16 rows of 128 B (128-byte swizzle), i.e. a K-major operand tile whose
//   rows are pixels.  Out-of-range coordinates are zero-filled by the TMA unit: that IS the zero padding (R-42).
//   For a 3x3 source the box has R = 10 rows: the three vertical taps dy are the same tile read at row offset
//   dy * 16 (2 KB, a whole number of 1 KB swizzle atoms), so one 20 KB load feeds three K steps; the horizontal
//   taps dx are separate loads (a shift by one pixel is not swizzle-aligned).
// B operand: the layer's weights packed at uf_cmn_set_param time as [N][K] bf16 (K order = the loop order below),
//   2-D TMA boxes of 64 (K) x N.
// CTA PAIRS (cta_group::2): the two CTAs of a cluster form one 256-pixel MMA tile (each CTA's own 128-pixel tile as
//   its half of A) and each loads only HALF of every weight tile (N/2 rows): an M = 128 single-CTA MMA reads
//   4 KB (A) + 32 N bytes (B) of shared memory per N/2 cycles — 128 B/clk at N = 128, the port limit, next to the TMA
//   writes — and ingests the whole weight tile per SM; in a pair it is 4 KB + 16 N bytes.  The leader CTA issues all
//   MMAs, TMA loads of both CTAs signal the leader's barriers, tcgen05.commit frees stages in both.
// A pair works on MT such double tiles at once so that every weight tile is loaded once per MT tiles: the L2 -> SM
//   path (about 42 B/clk/SM) is what bounds a tile with K = 64 per step otherwise.
// Warps: 0 = TMA producer, 1 = MMA issuer (+ TMEM allocation), 2..5 = epilogue (TMEM -> registers -> + bias,
//   ReLU, bf16 -> global, with the PixelShuffle / channel-to-time scatter folded into the store address).
//   Accumulators are double-buffered in TMEM when MT * N <= 256 columns.
#include "uf_cmn.h"
#include "uf_sm100_ptx.h"

#include <cuda_bf16.h>

#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace ufcmn {

using namespace ufptx;

constexpr int kConvThreads = 192;
constexpr int kATileBytes = 10 * 16 * 128;      // one tall A tile: 10 rows x 16 pixels x 64 channels bf16
constexpr int kMaxBias = 1024;                  // fp32 bias of one layer in shared memory
constexpr int kMaxSrc = 2;

enum OutMode { OUT_PLAIN = 0, OUT_SHUFFLE = 1, OUT_TEXP = 2 };

struct ConvParams {
  int n_src;
  int ntx[kMaxSrc], nty[kMaxSrc];   // taps of each source along x / y (3 or 1)
  int cchunks[kMaxSrc];             // 64-channel slices of each source
  int fbase[kMaxSrc];               // frame slot of output frame f in the source buffer = fbase + f ...
  int mem[kMaxSrc];                 // ... or, for a memory source, fbase + f - 1, and f0_slot for f == 0
  int f0_slot[kMaxSrc];
  int F, H, W;                      // frames of this launch, conv grid (= source grid)
  int tiles_x, tiles_y;             // 128-pixel tiles per frame: 8 rows x 16 columns each
  int n_ntiles, N;                  // N tiles, GEMM columns per tile (multiple of 16, <= 256)
  int nA, nB;                       // ring depths
  int n_acc;                        // accumulator buffers in TMEM (1 or 2)
  // output
  __nv_bfloat16* out;
  const float* bias;                // [n_ntiles * N]
  int n_total;                      // n_ntiles * N
  int relu;
  int mode, r, fs;                  // OutMode; PixelShuffle factor; frames per input frame (channel-to-time)
  int c_grp;                        // columns per output group (C for shuffle / texp, n_total for plain)
  int c_real;                       // columns of a group that exist in the output tensor
  int out_fbase;                    // frame slot offset in the output buffer
  int Hout, Wout, Cbuf;             // output tensor geometry (rows, columns, channel stride)
};

template <int MT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kConvThreads, 1)
uf_cmn_conv_kernel(const __grid_constant__ CUtensorMap tm_a0, const __grid_constant__ CUtensorMap tm_a1,
                   const __grid_constant__ CUtensorMap tm_b, const ConvParams p) {
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* base_ptr = smem_raw + (base - raw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  const uint32_t a_stage_bytes = MT * kATileBytes;
  const uint32_t b_stage_bytes = (uint32_t)(p.N / 2) * 128u;     // this CTA's half of the weight tile
  const uint32_t rank = cluster_ctarank();                        // 0 = leader of the pair
  const int pair = (int)(blockIdx.x >> 1), n_pairs = (int)(gridDim.x >> 1);
  const uint32_t off_b = p.nA * a_stage_bytes;
  const uint32_t off_bias = off_b + p.nB * b_stage_bytes;
  const uint32_t off_bar = off_bias + kMaxBias * 4;
  // barriers: A_FULL[nA] A_EMPTY[nA] B_FULL[nB] B_EMPTY[nB] ACC_FULL[2] ACC_EMPTY[2]
  const uint32_t bars = base + off_bar;
  const uint32_t bA_FULL = bars, bA_EMPTY = bars + 8 * p.nA, bB_FULL = bars + 16 * p.nA,
                 bB_EMPTY = bB_FULL + 8 * p.nB, bACC_FULL = bB_FULL + 16 * p.nB, bACC_EMPTY = bACC_FULL + 16;
  volatile uint32_t* tmem_ptr_smem = reinterpret_cast<volatile uint32_t*>(base_ptr + off_bar + 8 * (2 * p.nA + 2 * p.nB + 4));
  float* bias_s = reinterpret_cast<float*>(base_ptr + off_bias);

  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_a0));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_a1));
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_b));
    for (int i = 0; i < 2 * p.nA + 2 * p.nB + 2; ++i) mbar_init(bars + 8 * i, 1);
    mbar_init(bACC_EMPTY, 8);                          // the 4 epilogue warps of BOTH CTAs arrive on the leader's
    mbar_init(bACC_EMPTY + 8, 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32((const void*)tmem_ptr_smem)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  for (int i = threadIdx.x; i < p.n_total; i += kConvThreads) bias_s[i] = p.bias[i];
  tc_fence_before();
  __syncthreads();
  cluster_sync();                                      // the peer's barriers exist before anything signals them
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_smem;

  // Work = cells (N tile nt, double tile di = pixel tiles 2 di and 2 di + 1, one per CTA of the pair), nt outer; a pair
  // owns the contiguous range [cell_lo, cell_hi) of a balanced split and walks it in groups of up to MT double
  // tiles that share nt (and so every weight tile).  A pixel tile past the end (odd count) is all zero-fill.
  const int tiles_per_frame = p.tiles_x * p.tiles_y;
  const int m_tiles = p.F * tiles_per_frame;
  const int d_tiles = (m_tiles + 1) / 2;
  const int n_cells = d_tiles * p.n_ntiles;
  const int cq = n_cells / n_pairs, cr = n_cells % n_pairs;
  const int cell_lo = pair * cq + min(pair, cr);
  const int cell_hi = cell_lo + cq + (pair < cr ? 1 : 0);
  const uint32_t acc_stride = (p.n_acc == 2) ? 256u : 0u;

#define UF_GROUP_LOOP_BEGIN                                                                 \
  for (int cell = cell_lo; cell < cell_hi;) {                                               \
    const int nt = cell / d_tiles;                                                          \
    const int m0 = cell - nt * d_tiles;                                                     \
    const int cnt = min(MT, min(cell_hi - cell, d_tiles - m0));
#define UF_GROUP_LOOP_END cell += cnt; }
  // pixel tile mi -> frame, first row, first column
#define UF_MTILE_DECODE(mi)                                   \
  const int f = (mi) / tiles_per_frame;                       \
  const int rem = (mi) - f * tiles_per_frame;                 \
  const int y0 = (rem / p.tiles_x) * 8;                       \
  const int x0 = (rem % p.tiles_x) * 16;

  // programmatic dependent launch: everything above (barriers, TMEM, bias) overlapped the previous layer's tail;
  // from here on this grid reads what that layer wrote and overwrites buffers it may still read
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == 0) {
    // ================================ TMA producer ================================
    uint32_t as = 0, aph = 0, bs = 0, bph = 0;
    UF_GROUP_LOOP_BEGIN
      int kstep = 0;
      for (int s = 0; s < p.n_src; ++s) {
        const CUtensorMap* ta = s == 0 ? &tm_a0 : &tm_a1;
        const int ntx = p.ntx[s], nty = p.nty[s];
        const uint32_t a_bytes = (uint32_t)(nty == 3 ? 10 : 8) * 16u * 128u;
        for (int cc = 0; cc < p.cchunks[s]; ++cc) {
          for (int dxi = 0; dxi < ntx; ++dxi) {
            mbar_wait(bA_EMPTY + 8 * as, aph ^ 1);
            if (elect_one()) {
              if (rank == 0) mbar_expect_tx(bA_FULL + 8 * as, 2 * cnt * a_bytes);      // both CTAs' bytes
              for (int mt = 0; mt < cnt; ++mt) {
                UF_MTILE_DECODE(2 * (m0 + mt) + (int)rank)                                // past the end: frame out of range
                tma_load_4d_2sm(base + as * a_stage_bytes + mt * kATileBytes, ta, bA_FULL + 8 * as, cc * 64,
                                x0 + dxi - (ntx == 3 ? 1 : 0), y0 - (nty == 3 ? 1 : 0),
                                f >= p.F ? 0x100000 : !p.mem[s] ? p.fbase[s] + f : f ? p.fbase[s] + f - 1 : p.f0_slot[s]);
              }
            }
            if (++as == (uint32_t)p.nA) { as = 0; aph ^= 1; }
            for (int dyi = 0; dyi < nty; ++dyi) {
              mbar_wait(bB_EMPTY + 8 * bs, bph ^ 1);
              if (elect_one()) {
                if (rank == 0) mbar_expect_tx(bB_FULL + 8 * bs, 2 * b_stage_bytes);
                tma_load_2d_2sm(base + off_b + bs * b_stage_bytes, &tm_b, bB_FULL + 8 * bs, kstep * 64,
                                nt * p.N + (int)rank * (p.N / 2));
              }
              ++kstep;
              if (++bs == (uint32_t)p.nB) { bs = 0; bph ^= 1; }
            }
          }
        }
      }
    UF_GROUP_LOOP_END
  } else if (warp == 1) {
    // ================================ MMA issuer (leader CTA only) ================
    // instruction descriptor kind::f16: D fp32, A/B bf16 K-major, M = 256 over the pair, N = p.N
    const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (((uint32_t)p.N >> 3) << 17) | ((256u >> 4) << 24);
    if (rank == 0) {
    uint32_t as = 0, aph = 0, bs = 0, bph = 0, ab = 0, abph = 0;
    UF_GROUP_LOOP_BEGIN
      (void)nt;
      mbar_wait(bACC_EMPTY + 8 * ab, abph ^ 1);          // the epilogue has drained this accumulator buffer
      tc_fence_after();
      const uint32_t d_base = tmem + ab * acc_stride;
      bool first = true;
      for (int s = 0; s < p.n_src; ++s) {
        const int ntx = p.ntx[s], nty = p.nty[s];
        for (int cc = 0; cc < p.cchunks[s]; ++cc) {
          for (int dxi = 0; dxi < ntx; ++dxi) {
            mbar_wait(bA_FULL + 8 * as, aph);
            const uint32_t a_lo0 = desc_lo(base + as * a_stage_bytes);
            for (int dyi = 0; dyi < nty; ++dyi) {
              mbar_wait(bB_FULL + 8 * bs, bph);
              tc_fence_after();
              if (elect_one()) {
                const uint32_t b_lo = desc_lo(base + off_b + bs * b_stage_bytes);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                  if (mt >= cnt) break;
                  const uint32_t a_lo = a_lo0 + ((mt * kATileBytes + dyi * 2048) >> 4);
#pragma unroll
                  for (int k = 0; k < 4; ++k)             // 64 channels = 4 MMAs of K = 16 (32 B along the row)
                    mma_ss_2sm(d_base + mt * p.N, a_lo + k * 2, b_lo + k * 2, idesc, (first && k == 0) ? 0u : 1u);
                }
                tc_commit_2sm(bB_EMPTY + 8 * bs);
              }
              first = false;
              if (++bs == (uint32_t)p.nB) { bs = 0; bph ^= 1; }
            }
            if (elect_one()) tc_commit_2sm(bA_EMPTY + 8 * as);
            if (++as == (uint32_t)p.nA) { as = 0; aph ^= 1; }
          }
        }
      }
      if (elect_one()) tc_commit_2sm(bACC_FULL + 8 * ab);
      if (p.n_acc == 2) { if (++ab == 2) { ab = 0; abph ^= 1; } } else abph ^= 1;
    UF_GROUP_LOOP_END
    }
  } else {
    // ================================== epilogue ==================================
    const int q = warp & 3;                              // TMEM lane quarter this warp may access
    const int row = q * 32 + lane;                       // pixel of the tile == TMEM lane
    const int yy = row >> 4, xx = row & 15;
    const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
    uint32_t ab = 0, abph = 0;
    UF_GROUP_LOOP_BEGIN
      mbar_wait(bACC_FULL + 8 * ab, abph);
      tc_fence_after();
#pragma unroll 1
      for (int mt = 0; mt < cnt; ++mt) {
        UF_MTILE_DECODE(2 * (m0 + mt) + (int)rank)
        const int y = y0 + yy, x = x0 + xx;
        const bool valid = (f < p.F) && (y < p.H) && (x < p.W);
        const uint32_t t_base = tmem + lane_addr + ab * acc_stride + mt * p.N;
#pragma unroll 1
        for (int c0 = 0; c0 < p.N; c0 += 16) {
          uint32_t v[16];
          UFPTX_TMEM_LD16(t_base + c0, v);
          UFPTX_TMEM_WAIT_LD16(v);
          const int n0 = nt * p.N + c0;                  // global GEMM column of v[0]
          const int grp = n0 / p.c_grp, c = n0 - grp * p.c_grp;
          if (valid && c < p.c_real) {
            int fo = f * p.fs + p.out_fbase, yo = y * p.r, xo = x * p.r;
            if (p.mode == OUT_SHUFFLE) { yo += grp / p.r; xo += grp % p.r; }
            else if (p.mode == OUT_TEXP) fo += grp;
            __nv_bfloat16* dst = p.out + (((int64_t)fo * p.Hout + yo) * p.Wout + xo) * p.Cbuf + c;
            float o[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              o[j] = __uint_as_float(v[j]) + bias_s[n0 + j];
              if (p.relu) o[j] = fmaxf(o[j], 0.f);
            }
            if (c + 16 <= p.c_real && (p.Cbuf & 7) == 0) {
              uint4 w0, w1;
              w0.x = pack_bf16x2(o[0], o[1]);   w0.y = pack_bf16x2(o[2], o[3]);
              w0.z = pack_bf16x2(o[4], o[5]);   w0.w = pack_bf16x2(o[6], o[7]);
              w1.x = pack_bf16x2(o[8], o[9]);   w1.y = pack_bf16x2(o[10], o[11]);
              w1.z = pack_bf16x2(o[12], o[13]); w1.w = pack_bf16x2(o[14], o[15]);
              reinterpret_cast<uint4*>(dst)[0] = w0;
              reinterpret_cast<uint4*>(dst)[1] = w1;
            } else {
#pragma unroll
              for (int j = 0; j < 16; ++j)
                if (c + j < p.c_real) dst[j] = __float2bfloat16_rn(o[j]);
            }
          }
          __syncwarp();                                  // the TMEM loads are warp-collective (.aligned)
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_leader(bACC_EMPTY + 8 * ab);
      if (p.n_acc == 2) { if (++ab == 2) { ab = 0; abph ^= 1; } } else abph ^= 1;
    UF_GROUP_LOOP_END
  }
#undef UF_GROUP_LOOP_BEGIN
#undef UF_GROUP_LOOP_END
#undef UF_MTILE_DECODE

  tc_fence_before();
  __syncthreads();
  cluster_sync();                                      // neither CTA frees TMEM or exits while the other may still use it
  if (warp == 1) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
PFN_encodeTiled encode_fn() {
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

// activations bf16 [F][H][W][C]; box = 64 channels x 16 columns x box_rows rows x 1 frame (C < 64: the rest of the
// box is out of range and zero-filled)
bool encode_act_map(CUtensorMap* m, const void* ptr, int F, int H, int W, int C, int box_rows) {
  PFN_encodeTiled fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)C, (cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)F};
  const cuuint64_t strides[3] = {(cuuint64_t)C * 2, (cuuint64_t)W * C * 2, (cuuint64_t)H * W * C * 2};
  const cuuint32_t box[4] = {64, 16, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// weights bf16 [N][K]; box = 64 (K) x n_tile rows
bool encode_w_map(CUtensorMap* m, const void* ptr, int N, int K, int n_tile) {
  PFN_encodeTiled fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)N};
  const cuuint64_t strides[1] = {(cuuint64_t)K * 2};
  const cuuint32_t box[2] = {64, (cuuint32_t)n_tile};
  const cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct Buf {
  __nv_bfloat16* p = nullptr;
  int H = 0, W = 0, C = 0;
  int fmul = 1;              // frames per input frame at this point of the network
  // A block input keeps its own past (R-41): slot 0 is all zeros (the memory at the start of a stream), then two
  // regions of frames_max * fmul slots that successive steps fill in turn; the memory of a step is the slot the
  // previous step wrote its last frame to.  No copies: "memory" is the same tensor map at another frame coordinate.
  int has_mem = 0;
  int slots = 0;             // frame slots allocated: frames_max * fmul, or 1 + 2 * that
  int region = 0;            // region the NEXT step writes (has_mem only)
  int mem_slot = 0;          // slot of the current memory frame (0 = zeros)
  int last_base = 0;         // first slot the last step wrote
  int base(int frames_max) const { return has_mem ? 1 + region * frames_max * fmul : 0; }
  size_t frame_elems() const { return (size_t)H * W * C; }
};

struct Param {               // one parameter tensor as the caller names it
  std::string name;
  int shape[4];              // Cout, Cin, kh, kw
  int has_bias;
  int layer;                 // layer whose GEMM matrix it fills
  int src;                   // source index inside that layer
  int src_ci0;               // first input channel of that source within this tensor's Cin (c1: memory half = C)
  bool set = false;
};

struct Layer {
  std::string name;
  int n_src = 1;
  int src_buf[kMaxSrc] = {-1, -1};    // -1 = the caller's z
  int ntap[kMaxSrc] = {9, 9};         // 9 or 1
  int cin[kMaxSrc] = {0, 0};          // real channels of the source
  int mem[kMaxSrc] = {0, 0};          // 1: read one frame earlier
  int koff[kMaxSrc] = {0, 0};         // first K index of the source
  int cout = 0;                       // real GEMM columns
  int n_total = 0, n_tile = 0, n_ntiles = 1, K = 0, MT = 1;
  int relu = 0, mode = OUT_PLAIN, r = 1, fs = 1, c_grp = 0, c_real = 0;
  int out_buf = -1;                   // -1 = the caller's out
  int H = 0, W = 0, fmul = 1;         // conv grid, frames per input frame
  __nv_bfloat16* w = nullptr;         // device [n_total][K]
  float* bias = nullptr;              // device [n_total]
  CUtensorMap tm_a[kMaxSrc];
  // the N tile is chosen per step from up to two options (n_total split into k or 2k tiles), each with its own
  // weight tensor map
  int n_opt = 1, opt_ntile[2] = {0, 0};
  CUtensorMap tm_b[2];
  int opt = 0;                        // option of the current plan
  int plan_frames = -1;               // frames the current plan was made for
  int nA = 2, nB = 4, n_acc = 1;
  size_t smem = 0;
  int64_t flops_per_frame = 0;        // of one INPUT frame of the network
};

}  // namespace ufcmn

using namespace ufcmn;

struct uf_cmn {
  uf_cmn_config cfg;
  std::vector<Buf> bufs;
  std::vector<Layer> layers;
  std::vector<Param> params;
  std::vector<int> mem_buf;           // [stage * n_blocks + block] -> buffer holding that block's input
  int out_H = 0, out_W = 0, out_fmul = 1;
  int sm_count = 0;
  int64_t dev_bytes = 0, launches = 0;
  // tensor map of the caller's z for the input layer, re-encoded when (pointer, frames) change
  const void* z_ptr = nullptr;
  int z_frames = 0;
  int last_frames = 0;                // input frames of the last uf_cmn_step
  bool smem_attr[3] = {};             // 227 KB dynamic-smem limit already raised on uf_cmn_conv_kernel<1 | 2 | 4> for
                                      // THIS handle's device (the attribute is per device, so the flag is per handle)
  std::string err;
};

namespace {

thread_local std::string g_cmn_create_err;

int cfail(uf_cmn* n, int code, const std::string& msg) {
  if (n) n->err = msg; else g_cmn_create_err = msg;
  return code;
}

int stage_out_width(const uf_cmn_config& c, int s) {
  if (s + 1 < c.n_stages) return c.stage_channels[s + 1];
  return c.stage_channels[c.n_stages] > 0 ? c.stage_channels[c.n_stages] : c.stage_channels[s];
}

int add_buf(uf_cmn* n, int H, int W, int C, int fmul, int has_mem) {
  Buf b;
  b.H = H; b.W = W; b.C = C; b.fmul = fmul; b.has_mem = has_mem;
  b.slots = has_mem ? 1 + 2 * n->cfg.frames_max * fmul : n->cfg.frames_max * fmul;
  n->bufs.push_back(b);
  return (int)n->bufs.size() - 1;
}

// N tile, pixel tiles per group (MT) and ring depths of a layer for `frames` frames on `sms` SMs.
// Cost of an option = cells of the busiest CTA pair x columns per cell x a relative cost per column: per MMA a CTA
// of a pair reads 4 KB of A and 16 N bytes of B from shared memory per N/2 tensor cycles, i.e. 64 B/clk at N = 256,
// 96 at N = 128, 160 at N = 64 (above the 128 B/clk port), next to the TMA writes.  Narrower tiles only pay where
// they remove a whole round of CTA pairs.
double col_cost(int n_tile) { return n_tile > 128 ? 1.0 : n_tile > 64 ? 1.15 : 1.6; }

void plan_layer(Layer& L, int frames, int sms) {
  const int m_tiles = frames * ((L.H + 7) / 8) * ((L.W + 15) / 16);
  const int d_tiles = (m_tiles + 1) / 2, pairs = sms / 2;
  double best = 1e300;
  for (int o = 0; o < L.n_opt; ++o) {
    const int nt = L.opt_ntile[o], n_ntiles = L.n_total / nt;
    const int cells = d_tiles * n_ntiles;
    const int grid = cells < pairs ? cells : pairs;
    const int per_pair = (cells + grid - 1) / grid;
    const double cost = per_pair * (double)nt * col_cost(nt);
    if (cost < best) { best = cost; L.opt = o; }
  }
  L.n_tile = L.opt_ntile[L.opt];
  L.n_ntiles = L.n_total / L.n_tile;
  // Groups small enough for two accumulator buffers (MT * N <= 256 TMEM columns) let the epilogue of a group run under
  // the next group's main loop.  Exception (measured, r2e launch lists): when ALL cells of the busiest pair fit one
  // single-buffered group (MT * N <= 512), that one group — every weight tile loaded once — beats several small ones.
  {
    const int cells = ((m_tiles + 1) / 2) * L.n_ntiles;
    const int grid = cells < sms / 2 ? cells : sms / 2;
    const int per_pair = (cells + grid - 1) / grid;
    const int mt_single = L.n_tile > 128 ? 2 : 4, mt_double = L.n_tile > 128 ? 1 : L.n_tile > 64 ? 2 : 4;   // (N <= 64 with MT = 2 and a 4-deep A ring: measured slower)
    L.MT = per_pair <= mt_single ? mt_single : mt_double;
  }
  L.n_acc = (L.MT * L.n_tile <= 256) ? 2 : 1;
  // ring depths: an A stage (MT tall tiles) lasts 3 * 4 * MT * N/2 tensor cycles, less than a TMA round trip for the
  // narrow layers, so the A ring gets up to 4 stages once 6 weight stages (two (slice, dx) groups) are reserved
  const size_t budget = 227 * 1024 - 1024 - kMaxBias * 4 - 256;
  const size_t b_stage = (size_t)(L.n_tile / 2) * 128, a_stage = (size_t)L.MT * kATileBytes;
  int na = (int)((budget - 6 * b_stage) / a_stage);
  L.nA = na < 2 ? 2 : na > 4 ? 4 : na;
  const size_t a = (size_t)L.nA * a_stage;
  const int nb = (int)((budget - a) / b_stage);
  L.nB = nb > 8 ? 8 : nb;
  L.smem = a + (size_t)L.nB * (L.n_tile / 2) * 128 + kMaxBias * 4 + 256 + 1024;
  L.plan_frames = frames;
}

// the N-tile options of a layer: n_total in the fewest equal tiles of <= 256 columns, and twice as many
void tile_options(Layer& L) {
  int k = (L.n_total + 255) / 256;
  while (L.n_total % (16 * k)) ++k;
  L.opt_ntile[0] = L.n_total / k;
  L.n_opt = 1;
  if (L.opt_ntile[0] % 32 == 0 && L.opt_ntile[0] / 2 >= 64) {
    // halves must not cut a PixelShuffle / channel-to-time group of c_grp columns in an epilogue chunk: both are
    // multiples of 16, which is all the epilogue needs
    L.opt_ntile[1] = L.opt_ntile[0] / 2;
    L.n_opt = 2;
  }
}

template <int MT>
cudaError_t launch_conv(const Layer& L, const ConvParams& p, int grid, cudaStream_t s, bool& attr_set) {
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(uf_cmn_conv_kernel<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  // programmatic dependent launch: the next layer's prologue (barrier init, TMEM allocation, bias load) may start
  // while this layer's last CTAs finish; the kernel waits (griddepcontrol.wait) before it touches activations
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(kConvThreads); cfg.dynamicSmemBytes = L.smem; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, uf_cmn_conv_kernel<MT>, L.tm_a[0], L.tm_a[L.n_src > 1 ? 1 : 0], L.tm_b[L.opt], p);
}

void build_graph(uf_cmn* n) {
  const uf_cmn_config& c = n->cfg;
  int H = c.height, W = c.width, fmul = 1;
  auto conv = [&](const std::string& name, int src, int ntap, int cin, int cout, int out_buf) -> Layer& {
    Layer L;
    L.name = name;
    L.src_buf[0] = src; L.ntap[0] = ntap; L.cin[0] = cin; L.cout = cout;
    L.c_grp = 0; L.H = H; L.W = W; L.fmul = fmul; L.out_buf = out_buf;
    n->layers.push_back(L);
    return n->layers.back();
  };
  auto add_param = [&](const std::string& name, int co, int ci, int k, int has_bias, int layer, int src, int ci0) {
    Param p;
    p.name = name; p.shape[0] = co; p.shape[1] = ci; p.shape[2] = k; p.shape[3] = k;
    p.has_bias = has_bias; p.layer = layer; p.src = src; p.src_ci0 = ci0;
    n->params.push_back(p);
  };
  int C = c.stage_channels[0];
  int h = add_buf(n, H, W, C, fmul, 1);                               // input of s0.b0
  conv("in", -1, 9, c.in_ch, C, h);
  add_param("in", C, c.in_ch, 3, 1, 0, 0, 0);
  n->mem_buf.assign((size_t)c.n_stages * c.n_blocks, -1);
  for (int s = 0; s < c.n_stages; ++s) {
    C = c.stage_channels[s];
    for (int b = 0; b < c.n_blocks; ++b) {
      const std::string pre = "s" + std::to_string(s) + ".b" + std::to_string(b) + ".";
      // every layer keeps its own output buffer (observable through uf_cmn_get_activation)
      const int t1 = add_buf(n, H, W, C, fmul, 0), t2 = add_buf(n, H, W, C, fmul, 0);
      n->mem_buf[(size_t)s * c.n_blocks + b] = h;
      const int nxt = add_buf(n, H, W, C, fmul, b + 1 < c.n_blocks ? 1 : 0);
      {
        Layer& L = conv(pre + "c1", h, 9, C, C, t1);
        L.n_src = 2; L.src_buf[1] = h; L.ntap[1] = 9; L.cin[1] = C; L.mem[1] = 1; L.relu = 1;
        add_param(pre + "c1", C, 2 * C, 3, 1, (int)n->layers.size() - 1, -1, 0);    // src -1: both halves
      }
      conv(pre + "c2", t1, 9, C, C, t2);
      add_param(pre + "c2", C, C, 3, 1, (int)n->layers.size() - 1, 0, 0);
      {
        Layer& L = conv(pre + "c3+skip", t2, 9, C, C, nxt);
        L.n_src = 2; L.src_buf[1] = h; L.ntap[1] = 1; L.cin[1] = C; L.relu = 1;
        add_param(pre + "c3", C, C, 3, 1, (int)n->layers.size() - 1, 0, 0);
        add_param(pre + "skip", C, C, 1, 0, (int)n->layers.size() - 1, 1, 0);
      }
      h = nxt;
    }
    const int r = c.spatial_factors[s], ts = c.temporal_factors[s];
    const std::string pre = "s" + std::to_string(s) + ".";
    const int up = add_buf(n, H * r, W * r, C, fmul, 0);
    {
      Layer& L = conv(pre + "up", h, 9, C, C * r * r, up);
      if (r > 1) { L.mode = OUT_SHUFFLE; L.r = r; L.c_grp = C; }
      add_param(pre + "up", C * r * r, C, 3, 1, (int)n->layers.size() - 1, 0, 0);
    }
    H *= r; W *= r;
    h = up;
    if (ts > 1) {
      const int te = add_buf(n, H, W, C, fmul * ts, 0);
      Layer& L = conv(pre + "texp", h, 1, C, C * ts, te);
      L.mode = OUT_TEXP; L.fs = ts; L.c_grp = C;
      add_param(pre + "texp", C * ts, C, 1, 1, (int)n->layers.size() - 1, 0, 0);
      fmul *= ts;
      h = te;
    }
    const int Cn = stage_out_width(c, s);
    const int nb = add_buf(n, H, W, Cn, fmul, s + 1 < c.n_stages ? 1 : 0);
    {
      Layer& L = conv(pre + "ch", h, 1, C, Cn, nb);
      L.fmul = fmul;
      add_param(pre + "ch", Cn, C, 1, 1, (int)n->layers.size() - 1, 0, 0);
    }
    h = nb;
  }
  const int Cl = stage_out_width(c, c.n_stages - 1);
  {
    Layer& L = conv("out", h, 9, Cl, c.out_ch, -1);
    L.fmul = fmul;
    add_param("out", c.out_ch, Cl, 3, 1, (int)n->layers.size() - 1, 0, 0);
  }
  n->out_H = H; n->out_W = W; n->out_fmul = fmul;
  // derived GEMM shapes
  for (Layer& L : n->layers) {
    int k = 0;
    for (int s = 0; s < L.n_src; ++s) {
      L.koff[s] = k;
      k += L.ntap[s] * ((L.cin[s] + 63) / 64) * 64;
    }
    L.K = k;
    L.n_total = (L.cout + 15) / 16 * 16;
    if (L.c_grp == 0) { L.c_grp = L.n_total; L.c_real = L.cout; } else L.c_real = L.c_grp;
    tile_options(L);
    int64_t macs = 0;
    for (int s = 0; s < L.n_src; ++s) macs += (int64_t)L.ntap[s] * L.cin[s] * L.cout;
    // pixels of this layer per input frame of the network
    L.flops_per_frame = 2 * macs * L.H * L.W * L.fmul;
  }
}

bool supported(const uf_cmn_config& c, std::string* why) {
  auto bad = [&](const char* m) { *why = m; return false; };
  if (c.n_stages < 1 || c.n_stages > UF_CMN_MAX_STAGES) return bad("n_stages outside 1..4");
  if (c.n_blocks < 1 || c.n_blocks > 16) return bad("n_blocks outside 1..16");
  if (c.in_ch < 8 || c.in_ch > 64 || (c.in_ch % 8)) return bad("in_ch must be a multiple of 8, <= 64");
  if (c.out_ch < 1 || c.out_ch > 64) return bad("out_ch outside 1..64");
  if (c.height < 1 || c.width < 1 || c.frames_max < 1) return bad("height, width, frames_max must be >= 1");
  for (int s = 0; s <= c.n_stages; ++s) {
    const int C = c.stage_channels[s];
    if (s == c.n_stages && C == 0) continue;
    if (C < 64 || C > 256 || (C % 64)) return bad("stage_channels must be multiples of 64 in 64..256");
  }
  for (int s = 0; s < c.n_stages; ++s) {
    if (c.spatial_factors[s] < 1 || c.spatial_factors[s] > 3) return bad("spatial factor outside 1..3");
    if (c.temporal_factors[s] < 1 || c.temporal_factors[s] > 4) return bad("temporal factor outside 1..4");
    if (c.stage_channels[s] * c.spatial_factors[s] * c.spatial_factors[s] > kMaxBias)
      return bad("C * r^2 exceeds 1024 GEMM columns");
  }
  return true;
}

}  // namespace

extern "C" {

int32_t uf_cmn_create(const uf_cmn_config* cfg, uf_cmn** out) {
  if (!cfg || !out) return cfail(nullptr, UF_ERR_INVALID_ARG, "uf_cmn_create: null argument");
  std::string why;
  if (!supported(*cfg, &why)) return cfail(nullptr, UF_ERR_UNSUPPORTED, "uf_cmn_create: " + why);
  uf_cmn* n = new (std::nothrow) uf_cmn();
  if (!n) return cfail(nullptr, UF_ERR_CUDA, "uf_cmn_create: out of host memory");
  n->cfg = *cfg;
  build_graph(n);
  auto bail = [&](int code, const std::string& msg) {
    g_cmn_create_err = msg;
    uf_cmn_destroy(n);
    return code;
  };
  cudaError_t e = cudaSetDevice(cfg->device);
  if (e != cudaSuccess) return bail(UF_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, cfg->device);
  if (e != cudaSuccess) return bail(UF_ERR_CUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
  if (prop.major != 10) return bail(UF_ERR_UNSUPPORTED, "uf_cmn_create: the kernels are sm_100a only");
  n->sm_count = prop.multiProcessorCount;
  for (Buf& b : n->bufs) {
    const size_t bytes = b.frame_elems() * b.slots * sizeof(__nv_bfloat16);
    e = cudaMalloc(&b.p, bytes);
    if (e != cudaSuccess) return bail(UF_ERR_CUDA, std::string("cudaMalloc(activations): ") + cudaGetErrorString(e));
    n->dev_bytes += (int64_t)bytes;
    if (b.has_mem) {
      e = cudaMemset(b.p, 0, b.frame_elems() * sizeof(__nv_bfloat16));
      if (e != cudaSuccess) return bail(UF_ERR_CUDA, std::string("cudaMemset(memory): ") + cudaGetErrorString(e));
    }
  }
  for (Layer& L : n->layers) {
    const size_t wb = (size_t)L.n_total * L.K * sizeof(__nv_bfloat16);
    e = cudaMalloc(&L.w, wb);
    if (e == cudaSuccess) e = cudaMemset(L.w, 0, wb);
    if (e == cudaSuccess) e = cudaMalloc(&L.bias, (size_t)L.n_total * sizeof(float));
    if (e == cudaSuccess) e = cudaMemset(L.bias, 0, (size_t)L.n_total * sizeof(float));
    if (e != cudaSuccess) return bail(UF_ERR_CUDA, std::string("cudaMalloc(weights): ") + cudaGetErrorString(e));
    n->dev_bytes += (int64_t)wb + L.n_total * 4;
    for (int o = 0; o < L.n_opt; ++o)
      if (!encode_w_map(&L.tm_b[o], L.w, L.n_total, L.K, L.opt_ntile[o] / 2))      // a CTA loads half a tile
        return bail(UF_ERR_CUDA, "cuTensorMapEncodeTiled failed for the weights of " + L.name);
    for (int s = 0; s < L.n_src; ++s) {
      if (L.src_buf[s] < 0) continue;                       // the caller's z: encoded per step
      const Buf& b = n->bufs[L.src_buf[s]];
      if (!encode_act_map(&L.tm_a[s], b.p, b.slots, b.H, b.W, b.C, L.ntap[s] == 9 ? 10 : 8))
        return bail(UF_ERR_CUDA, "cuTensorMapEncodeTiled failed for a source of " + L.name);
    }
  }
  *out = n;
  return UF_OK;
}

int32_t uf_cmn_destroy(uf_cmn* n) {
  if (!n) return UF_OK;
  cudaSetDevice(n->cfg.device);
  for (Buf& b : n->bufs) if (b.p) cudaFree(b.p);
  for (Layer& L : n->layers) { if (L.w) cudaFree(L.w); if (L.bias) cudaFree(L.bias); }
  delete n;
  return UF_OK;
}

const char* uf_cmn_last_error(const uf_cmn* n) { return n ? n->err.c_str() : g_cmn_create_err.c_str(); }
int32_t uf_cmn_n_params(const uf_cmn* n) { return n ? (int32_t)n->params.size() : 0; }
int32_t uf_cmn_n_layers(const uf_cmn* n) { return n ? (int32_t)n->layers.size() : 0; }
int64_t uf_cmn_device_bytes(const uf_cmn* n) { return n ? n->dev_bytes : 0; }
int64_t uf_cmn_launches(const uf_cmn* n) { return n ? n->launches : 0; }

int32_t uf_cmn_param_info(const uf_cmn* n, int32_t index, char* name, int32_t name_cap, int32_t shape[4],
                          int32_t* has_bias) {
  if (!n || index < 0 || index >= (int32_t)n->params.size()) return UF_ERR_INVALID_ARG;
  const Param& p = n->params[index];
  if (name && name_cap > 0) snprintf(name, (size_t)name_cap, "%s", p.name.c_str());
  if (shape) for (int i = 0; i < 4; ++i) shape[i] = p.shape[i];
  if (has_bias) *has_bias = p.has_bias;
  return UF_OK;
}

int32_t uf_cmn_layer_info(const uf_cmn* n, int32_t index, char* name, int32_t name_cap, int64_t* flops_per_frame,
                          int32_t* gemm_n, int32_t* gemm_k, int32_t out_shape[4]) {
  if (!n || index < 0 || index >= (int32_t)n->layers.size()) return UF_ERR_INVALID_ARG;
  const Layer& L = n->layers[index];
  if (name && name_cap > 0) snprintf(name, (size_t)name_cap, "%s", L.name.c_str());
  if (flops_per_frame) *flops_per_frame = L.flops_per_frame;
  if (gemm_n) *gemm_n = L.n_total;
  if (gemm_k) *gemm_k = L.K;
  if (out_shape) {
    if (L.out_buf >= 0) {
      const Buf& b = n->bufs[L.out_buf];
      out_shape[0] = b.fmul; out_shape[1] = b.H; out_shape[2] = b.W; out_shape[3] = b.C;
    } else {
      out_shape[0] = n->out_fmul; out_shape[1] = n->out_H; out_shape[2] = n->out_W; out_shape[3] = n->cfg.out_ch;
    }
  }
  return UF_OK;
}

int64_t uf_cmn_flops(const uf_cmn* n, int32_t n_frames) {
  if (!n) return 0;
  int64_t t = 0;
  for (const Layer& L : n->layers) t += L.flops_per_frame;
  return t * n_frames;
}

int32_t uf_cmn_set_param(uf_cmn* n, const char* name, const void* w_host, const float* bias_host) {
  if (!n || !name || !w_host) return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_set_param: null argument");
  Param* pp = nullptr;
  for (Param& p : n->params) if (p.name == name) pp = &p;
  if (!pp) return cfail(n, UF_ERR_INVALID_ARG, std::string("uf_cmn_set_param: unknown parameter ") + name);
  if (!pp->has_bias && bias_host) return cfail(n, UF_ERR_INVALID_ARG, std::string(name) + " has no bias (R-43)");
  { cudaError_t de = cudaSetDevice(n->cfg.device);
    if (de != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(de)); }
  Layer& L = n->layers[pp->layer];
  const int Co = pp->shape[0], Ci = pp->shape[1], kk = pp->shape[2] * pp->shape[3];
  const uint16_t* w = static_cast<const uint16_t*>(w_host);
  // GEMM row of output channel o: PixelShuffle groups its r*r sub-pixels (i, j) into runs of C columns (R-44)
  auto row_of = [&](int o) {
    if (L.mode == OUT_SHUFFLE) { const int rr = L.r * L.r; return (o % rr) * L.c_grp + o / rr; }
    return o;
  };
  // read the layer's matrix back only when two tensors share it; simpler: keep a host mirror per call
  std::vector<uint16_t> mat((size_t)L.n_total * L.K);
  cudaError_t e = cudaMemcpy(mat.data(), L.w, mat.size() * 2, cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaMemcpy(weights D2H): ") + cudaGetErrorString(e));
  const int s_lo = pp->src < 0 ? 0 : pp->src, s_hi = pp->src < 0 ? L.n_src - 1 : pp->src;
  for (int s = s_lo; s <= s_hi; ++s) {
    const int ci0 = pp->src < 0 ? s * L.cin[0] : pp->src_ci0;
    const int ntap = L.ntap[s], cpad = (L.cin[s] + 63) / 64 * 64, cch = cpad / 64;
    const int ntx = ntap == 9 ? 3 : 1, nty = ntx;
    if (ntap != kk) return cfail(n, UF_ERR_INVALID_ARG, std::string(name) + ": kernel size does not match the layer");
    for (int o = 0; o < Co; ++o) {
      uint16_t* dst = mat.data() + (size_t)row_of(o) * L.K + L.koff[s];
      for (int cc = 0; cc < cch; ++cc)
        for (int dxi = 0; dxi < ntx; ++dxi)
          for (int dyi = 0; dyi < nty; ++dyi)
            for (int ci = 0; ci < 64; ++ci) {
              const int c = cc * 64 + ci;
              uint16_t v = 0;
              if (c < L.cin[s]) v = w[(((size_t)o * Ci + ci0 + c) * nty + dyi) * ntx + dxi];
              dst[((cc * ntx + dxi) * nty + dyi) * 64 + ci] = v;
            }
    }
  }
  e = cudaMemcpy(L.w, mat.data(), mat.size() * 2, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaMemcpy(weights H2D): ") + cudaGetErrorString(e));
  if (pp->has_bias) {
    std::vector<float> b((size_t)L.n_total, 0.f);
    if (bias_host) for (int o = 0; o < Co; ++o) b[row_of(o)] = bias_host[o];
    e = cudaMemcpy(L.bias, b.data(), b.size() * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaMemcpy(bias): ") + cudaGetErrorString(e));
  }
  pp->set = true;
  return UF_OK;
}

int32_t uf_cmn_reset(uf_cmn* n, void* stream) {
  if (!n) return UF_ERR_INVALID_ARG;
  (void)stream;
  // host state only: slot 0 of every block input is zero for good, and the next step takes it as its memory
  for (Buf& b : n->bufs) { b.mem_slot = 0; b.region = 0; }
  return UF_OK;
}

int32_t uf_cmn_step(uf_cmn* n, const void* z, int32_t n_frames, void* out, void* stream) {
  if (!n || !z || !out) return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_step: null argument");
  if (((uintptr_t)z & 15) || ((uintptr_t)out & 15)) return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_step: z and out must be 16-byte aligned");
  if (n_frames < 1 || n_frames > n->cfg.frames_max) return cfail(n, UF_ERR_CAPACITY, "uf_cmn_step: n_frames outside 1..frames_max");
  for (const Param& p : n->params)
    if (!p.set) return cfail(n, UF_ERR_STATE, "uf_cmn_step: parameter " + p.name + " was never set");
  { cudaError_t de = cudaSetDevice(n->cfg.device);
    if (de != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(de)); }
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const uf_cmn_config& c = n->cfg;
  if (n->z_ptr != z || n->z_frames != n_frames) {
    if (!encode_act_map(&n->layers[0].tm_a[0], z, n_frames, c.height, c.width, c.in_ch, 10))
      return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_step: cuTensorMapEncodeTiled failed for z");
    n->z_ptr = z; n->z_frames = n_frames;
  }
  for (Layer& L : n->layers) {
    if (L.plan_frames != n_frames * L.fmul) plan_layer(L, n_frames * L.fmul, n->sm_count);
    ConvParams p;
    memset(&p, 0, sizeof(p));
    p.n_src = L.n_src;
    for (int i = 0; i < L.n_src; ++i) {
      p.ntx[i] = p.nty[i] = L.ntap[i] == 9 ? 3 : 1;
      p.cchunks[i] = (L.cin[i] + 63) / 64;
      const Buf* sb = L.src_buf[i] >= 0 ? &n->bufs[L.src_buf[i]] : nullptr;
      p.fbase[i] = sb ? sb->base(c.frames_max) : 0;
      p.mem[i] = L.mem[i];
      p.f0_slot[i] = sb ? sb->mem_slot : 0;
    }
    p.F = n_frames * L.fmul; p.H = L.H; p.W = L.W;
    p.tiles_x = (L.W + 15) / 16;
    p.tiles_y = (L.H + 7) / 8;
    p.n_ntiles = L.n_ntiles; p.N = L.n_tile; p.nA = L.nA; p.nB = L.nB; p.n_acc = L.n_acc;
    p.bias = L.bias; p.n_total = L.n_total; p.relu = L.relu;
    p.mode = L.mode; p.r = L.r; p.fs = L.fs; p.c_grp = L.c_grp; p.c_real = L.c_real;
    if (L.out_buf >= 0) {
      const Buf& b = n->bufs[L.out_buf];
      p.out = b.p; p.out_fbase = b.base(c.frames_max); p.Hout = b.H; p.Wout = b.W; p.Cbuf = b.C;
    } else {
      p.out = static_cast<__nv_bfloat16*>(out); p.out_fbase = 0; p.Hout = n->out_H; p.Wout = n->out_W; p.Cbuf = c.out_ch;
    }
    const int n_cells = ((p.F * p.tiles_x * p.tiles_y + 1) / 2) * p.n_ntiles;      // (N tile, double pixel tile)
    const int pairs = n_cells < n->sm_count / 2 ? n_cells : n->sm_count / 2;
    const int grid = 2 * pairs;
    cudaError_t e = L.MT == 1 ? launch_conv<1>(L, p, grid, s, n->smem_attr[0])
                  : L.MT == 2 ? launch_conv<2>(L, p, grid, s, n->smem_attr[1])
                              : launch_conv<4>(L, p, grid, s, n->smem_attr[2]);
    if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, "uf_cmn_conv_kernel (" + L.name + "): " + cudaGetErrorString(e));
    ++n->launches;
  }
  n->last_frames = n_frames;
  // the last frame of every block input is the memory of the next step (R-41): remember where it is, switch regions
  for (Buf& b : n->bufs) {
    b.last_base = b.base(c.frames_max);
    if (b.has_mem) {
      b.mem_slot = b.last_base + n_frames * b.fmul - 1;
      b.region ^= 1;
    }
  }
  return UF_OK;
}

int32_t uf_cmn_get_memory(uf_cmn* n, int32_t stage, int32_t block, void* out_host, int32_t shape_out[3], void* stream) {
  if (!n || !out_host) return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_get_memory: null argument");
  if (stage < 0 || stage >= n->cfg.n_stages || block < 0 || block >= n->cfg.n_blocks)
    return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_get_memory: no such block");
  { cudaError_t de = cudaSetDevice(n->cfg.device);
    if (de != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(de)); }
  const Buf& b = n->bufs[n->mem_buf[(size_t)stage * n->cfg.n_blocks + block]];
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e = cudaMemcpyAsync(out_host, b.p + b.frame_elems() * (size_t)b.mem_slot, b.frame_elems() * sizeof(__nv_bfloat16),
                                  cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("uf_cmn_get_memory: ") + cudaGetErrorString(e));
  if (shape_out) { shape_out[0] = b.H; shape_out[1] = b.W; shape_out[2] = b.C; }
  return UF_OK;
}

int32_t uf_cmn_get_activation(uf_cmn* n, int32_t layer, void* out_host, int32_t shape_out[4], void* stream) {
  if (!n || !out_host) return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_get_activation: null argument");
  if (layer < 0 || layer >= (int32_t)n->layers.size() || n->layers[layer].out_buf < 0)
    return cfail(n, UF_ERR_INVALID_ARG, "uf_cmn_get_activation: no such layer (the last layer writes the caller's out)");
  if (n->last_frames < 1) return cfail(n, UF_ERR_STATE, "uf_cmn_get_activation: no step has run");
  { cudaError_t de = cudaSetDevice(n->cfg.device);
    if (de != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(de)); }
  const Buf& b = n->bufs[n->layers[layer].out_buf];
  const int F = n->last_frames * b.fmul;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e = cudaMemcpyAsync(out_host, b.p + b.frame_elems() * (size_t)b.last_base,
                                  b.frame_elems() * (size_t)F * sizeof(__nv_bfloat16), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return cfail(n, UF_ERR_CUDA, std::string("uf_cmn_get_activation: ") + cudaGetErrorString(e));
  if (shape_out) { shape_out[0] = F; shape_out[1] = b.H; shape_out[2] = b.W; shape_out[3] = b.C; }
  return UF_OK;
}

}  // extern "C"
