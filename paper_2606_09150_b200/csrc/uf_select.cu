// uf_select.cu — steps a2-a4: block-mean pooling of Q, block scores (Eq. 4) and exact
// top-k per (head, query block) with ties to the lower global id (BJ), plus the merge of the two
// lists of a query-block pair that the sm100 attention kernel walks.
//
// Arithmetic that decides indices is fp64 and follows the order stated in DESIGN.md R-4: the pooled
// sums are exact (order-free), the mean is one IEEE division, the dot product adds its d products in
// index order with separately rounded multiply and add (no FMA), then one IEEE division by sqrt(d).
#include "uf_internal.h"

namespace {

constexpr int kPoolThreads = 256;
constexpr int kScoreThreads = 256;

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// ---- a2: pooled Q.  grid (query blocks, H) -------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kPoolThreads)
uf_pool_q_kernel(const __nv_bfloat16* __restrict__ q, int64_t tok_stride, int64_t head_stride,
                 double* __restrict__ qbar, int B, int BPC, int ntok, UfTiling til) {
  constexpr int VPR = D / 8;
  constexpr int RPP = kPoolThreads / VPR;
  __shared__ double red[RPP][D + 2];
  const int i = blockIdx.x, h = blockIdx.y;
  const int vcx = threadIdx.x % VPR, rg = threadIdx.x / VPR;
  const int row0 = i * B;
  const int nvalid = til.enabled ? uf_tile_nvalid(til, i) : min(B, ntok - row0);
  double acc[8];
#pragma unroll
  for (int t = 0; t < 8; ++t) acc[t] = 0.0;
#pragma unroll 4
  for (int r = rg; r < nvalid; r += RPP) {
    const int64_t src = (int64_t)(row0 + r) * tok_stride + (int64_t)h * head_stride + vcx * 8;
    const uint4 u = ld_stream(reinterpret_cast<const uint4*>(q + src));
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      acc[2 * t]     += (double)__uint_as_float(w[t] << 16);
      acc[2 * t + 1] += (double)__uint_as_float(w[t] & 0xFFFF0000u);
    }
  }
#pragma unroll
  for (int t = 0; t < 8; ++t) red[rg][vcx * 8 + t] = acc[t];
  __syncthreads();
  if (threadIdx.x < D) {
    double s = 0.0;
#pragma unroll
    for (int g = 0; g < RPP; ++g) s += red[g][threadIdx.x];
    qbar[((int64_t)h * BPC + i) * D + threadIdx.x] = s / (double)nvalid;
  }
}

// order-preserving map double -> uint64 (no NaNs; -0.0 was normalised to +0.0 by the caller)
__device__ __forceinline__ unsigned long long sortable(double x) {
  unsigned long long u = (unsigned long long)__double_as_longlong(x);
  return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}

__device__ __forceinline__ void uf_merge_pair(const UfView& v, uint32_t* bma, uint32_t* bmb, int nw, int h, int p, int nqb,
                                              int k_eff, int kcap, const int32_t* __restrict__ sel_rank,
                                              const int32_t* __restrict__ sel_cnt, int32_t* __restrict__ sel_pair,
                                              int32_t* __restrict__ pair_cnt, int lane);

// ---- a3 + a4: scores and top-k.  grid (ceil(nqb / kQG), H) ------------------------------------------
// kQG query blocks are scored per CTA (each pooled-K load is re-used kQG times).
// dynamic smem: double qs[kQG][D]; unsigned long long key[kQG][n_cand]
// kPaper (Eq. 4 as written; R-32/R-33): the candidates are ALL blocks in the causal mask (the view lists the
// current chunk as its last "prior"), the top-k' is taken over all of them and THEN intersected with the r x r
// window M_local; the query block's own key block is always kept.  Rows then differ in length: sel_cnt holds
// each row's count and idx_out rows (out_stride entries) are padded with -1.
template <int D, int kQG, bool kPaper, int kPF>
__global__ void __launch_bounds__(kScoreThreads)
uf_score_topk_kernel(UfView v, const double* __restrict__ qbar, const double* __restrict__ kpool,
                     int nqb, int k_eff, int32_t* __restrict__ sel_q, int32_t* __restrict__ sel_rank, int kcap,
                     int32_t* __restrict__ sel_cnt, int32_t* __restrict__ idx_out, int32_t* __restrict__ cnt_out,
                     int out_stride, unsigned long long* __restrict__ usage,
                     int32_t* __restrict__ sel_pair, int32_t* __restrict__ pair_cnt,
                     unsigned long long* __restrict__ usage_next) {
  __shared__ unsigned int usage_s[UF_MAXC];            // kept blocks per listed chunk, this CTA (NEXT-3 statistic)
  if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x < UF_MAXC) usage_next[threadIdx.x] = 0ull;   // the next selection's
  if (threadIdx.x < UF_MAXC) usage_s[threadIdx.x] = 0u;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* qs = reinterpret_cast<double*>(smem_raw);                                  // [kQG][D]
  unsigned long long* key = reinterpret_cast<unsigned long long*>(qs + kQG * D);     // [kQG][n_cand]
  const int h = blockIdx.y;
  const int i0 = blockIdx.x * kQG;
  const int ng = min(kQG, nqb - i0);
  const int nc = v.n_cand;
  const int tid = threadIdx.x;

  for (int x = tid; x < kQG * D; x += kScoreThreads) {
    const int g = x / D, t = x % D;
    qs[x] = g < ng ? qbar[((int64_t)h * v.BPC + i0 + g) * D + t] : 0.0;
  }
  __syncthreads();

  const double inv = sqrt((double)D);
  for (int j = tid; j < nc; j += kScoreThreads) {
    int gid, phys, nval;
    uf_cand_lookup(v, j, &gid, &phys, &nval);
    const double* kp = kpool + (int64_t)h * D * v.P + phys;
    double acc[kQG];
#pragma unroll
    for (int g = 0; g < kQG; ++g) acc[g] = 0.0;
    // pooled-K loads run one batch of kPF ahead of the arithmetic (the loads are L2 hits ~700 cycles away; the dot
    // product itself is a dependent chain); the additions stay in index order (R-4)
    double kv[kPF], kn[kPF];
#pragma unroll
    for (int u = 0; u < kPF; ++u) kv[u] = __ldg(kp + (int64_t)u * v.P);
#pragma unroll 1
    for (int t0 = 0; t0 < D; t0 += kPF) {
      if (t0 + kPF < D) {
#pragma unroll
        for (int u = 0; u < kPF; ++u) kn[u] = __ldg(kp + (int64_t)(t0 + kPF + u) * v.P);
      }
#pragma unroll
      for (int u = 0; u < kPF; u += 2) {
#pragma unroll
        for (int g = 0; g < kQG; ++g) {
          const double2 q2 = *reinterpret_cast<const double2*>(qs + g * D + t0 + u);   // one 16-byte broadcast read
          acc[g] = __dadd_rn(acc[g], __dmul_rn(q2.x, kv[u]));
          acc[g] = __dadd_rn(acc[g], __dmul_rn(q2.y, kv[u + 1]));
        }
      }
#pragma unroll
      for (int u = 0; u < kPF; ++u) kv[u] = kn[u];
    }
#pragma unroll
    for (int g = 0; g < kQG; ++g) key[(int64_t)g * nc + j] = sortable(__ddiv_rn(acc[g], inv) + 0.0);
  }
  __syncthreads();

  // Exact top-k', one warp per query block.  T = a threshold with #{key > T} < k' <= #{key >= T}, found bit by
  // bit from the top (the largest value with #{key >= T} >= k').  Kept: every key > T, and of the keys == T the first
  // (k' - #{key > T}) in candidate order, i.e. ties go to the lower global id (R-12).  Candidates are in
  // ascending global id, so the ordered ballot compaction below emits ascending ids.
  const int lane = tid & 31, wid = tid >> 5;
  for (int g = wid; g < ng; g += kScoreThreads / 32) {
    const unsigned long long* kg = key + (int64_t)g * nc;
    const int i = i0 + g;
    // high words first (32 rounds on 32-bit values); the low words only matter if more keys share the high word
    // of the k'-th than may be kept (scores that agree to ~2^-20 relative: rare)
    const uint32_t* kw = reinterpret_cast<const uint32_t*>(kg);      // little endian: [2j] low, [2j + 1] high
    uint32_t Th = 0u;
    for (int b = 31; b >= 0; --b) {
      const uint32_t cand = Th | (1u << b);
      int cnt = 0;
      for (int j = lane; j < nc; j += 32) cnt += (kw[2 * j + 1] >= cand);
      cnt = __reduce_add_sync(0xffffffffu, cnt);
      if (cnt >= k_eff) Th = cand;
    }
    int c_gt = 0, c_eq = 0;
    for (int j = lane; j < nc; j += 32) { const uint32_t hw = kw[2 * j + 1]; c_gt += (hw > Th); c_eq += (hw == Th); }
    c_gt = __reduce_add_sync(0xffffffffu, c_gt);
    c_eq = __reduce_add_sync(0xffffffffu, c_eq);
    uint32_t Tl = 0u;                                 // c_gt + c_eq == k': every key with that high word is kept
    if (c_gt + c_eq > k_eff) {
      const int need = k_eff - c_gt;                  // of the keys with high word Th keep the `need` largest
      for (int b = 31; b >= 0; --b) {
        const uint32_t cand = Tl | (1u << b);
        int cnt = 0;
        for (int j = lane; j < nc; j += 32) cnt += (kw[2 * j + 1] == Th && kw[2 * j] >= cand);
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        if (cnt >= need) Tl = cand;
      }
    }
    const unsigned long long T = ((unsigned long long)Th << 32) | Tl;
    int n_gt = 0;
    for (int j = lane; j < nc; j += 32) n_gt += (kg[j] > T);
    n_gt = __reduce_add_sync(0xffffffffu, n_gt);
    const int need_eq = k_eff - n_gt;                  // keys == T still to keep (lowest candidate index first)
    int pos0 = 0, eq_seen = 0;
    const int64_t rowq = ((int64_t)h * v.BPC + i) * kcap;
    for (int j0 = 0; j0 < nc; j0 += 32) {
      const int j = j0 + lane;
      const unsigned long long mine = j < nc ? kg[j] : 0ull;
      const bool gt = j < nc && mine > T, eq = j < nc && mine == T;
      const unsigned beq = __ballot_sync(0xffffffffu, eq);
      bool keep = gt || (eq && eq_seen + __popc(beq & ((1u << lane) - 1u)) < need_eq);
      int gid = 0, phys = 0, nval = 1;
      if (kPaper && j < nc) {
        uf_cand_lookup(v, j, &gid, &phys, &nval);
        const int bj = gid % v.BPC;                    // block of its chunk (every chunk has the same tile grid)
        keep = (keep && uf_tile_local(v.til, i, bj)) || gid == v.cur_chunk * v.BPC + i;
      }
      const unsigned ball = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const int pos = pos0 + __popc(ball & ((1u << lane) - 1u));
        if (!kPaper) uf_cand_lookup(v, j, &gid, &phys, &nval);
        sel_q[rowq + pos] = uf_entry_pack(phys, nval, 0);
        sel_rank[rowq + pos] = j;                      // candidate index: the merge key
        if (idx_out) idx_out[((int64_t)h * nqb + i) * out_stride + pos] = gid;
        atomicAdd(&usage_s[uf_cand_prior(v, j)], 1u);
      }
      pos0 += __popc(ball);
      eq_seen += __popc(beq);
    }
    if (kPaper) {
      if (idx_out)
        for (int x = pos0 + lane; x < out_stride; x += 32) idx_out[((int64_t)h * nqb + i) * out_stride + x] = -1;
      if (lane == 0) sel_cnt[(int64_t)h * v.BPC + i] = pos0;
    }
    if (lane == 0 && cnt_out) cnt_out[(int64_t)h * nqb + i] = kPaper ? pos0 : k_eff;
  }
  __syncthreads();
  if (tid < v.n_prior && usage_s[tid]) atomicAdd(&usage[tid], (unsigned long long)usage_s[tid]);
  // Merge the lists of the query-block pairs this CTA just selected (kQG even, i0 a multiple of kQG: both blocks of
  // a pair are here; their sel_rank rows were written by this CTA before the barrier above) into the union lists
  // the tcgen05 attention kernels walk: no separate launch.  The key array is dead: its memory holds the bitmaps.
  if (sel_pair != nullptr && kQG >= 2) {
    const int nw = (nc + 31) / 32;
    uint32_t* bm = reinterpret_cast<uint32_t*>(key);
    for (int pp = wid; 2 * pp < ng; pp += kScoreThreads / 32)
      uf_merge_pair(v, bm + (size_t)pp * 2 * nw, bm + (size_t)pp * 2 * nw + nw, nw, h, i0 / 2 + pp, nqb, k_eff, kcap,
                    sel_rank, kPaper ? sel_cnt : nullptr, sel_pair, pair_cnt, lane);
  }
}

// ---- merge the lists of query blocks (2p, 2p+1) into one union list with tile masks -----------------
// One warp per (h, pair).  Both lists are subsets of CAND; sel_rank holds the candidate index of every kept
// entry, so each list becomes a bitmap over the candidates in shared memory.  Output order (the attention
// kernel's softmax does not depend on it): first the entries BOTH tiles attend (mask 3), then the entries only
// one tile attends, alternating tile 0 / tile 1 (mask 1, 2, 1, 2, ...), so that while one tile's softmax runs the
// tensor pipe has the other tile's MMAs (two single-tile steps of the same tile in a row would serialise).
// An entry's position is its rank within its class (word popcounts + a warp scan); its payload (physical
// block, valid rows) is recomputed from the candidate index.  dynamic smem: uint32 [warps][2][ceil(n_cand / 32)]
// One warp merges the lists of query blocks (2p, 2p + 1) of head h; bma / bmb: nw words of shared memory each.
__device__ __forceinline__ void uf_merge_pair(const UfView& v, uint32_t* bma, uint32_t* bmb, int nw, int h, int p, int nqb,
                                              int k_eff, int kcap, const int32_t* __restrict__ sel_rank,
                                              const int32_t* __restrict__ sel_cnt, int32_t* __restrict__ sel_pair,
                                              int32_t* __restrict__ pair_cnt, int lane) {
  const int NP = (v.BPC + 1) / 2;
  for (int w = lane; w < nw; w += 32) { bma[w] = 0u; bmb[w] = 0u; }
  __syncwarp();
  const int32_t* ra = sel_rank + ((int64_t)h * v.BPC + 2 * p) * kcap;
  const int32_t* rb = ra + kcap;
  const bool has1 = 2 * p + 1 < nqb;
  // rows of equal length k_eff (flat mode) or of their own length (paper-mask mode: sel_cnt)
  const int na = sel_cnt ? sel_cnt[(int64_t)h * v.BPC + 2 * p] : k_eff;
  const int nb = !has1 ? 0 : (sel_cnt ? sel_cnt[(int64_t)h * v.BPC + 2 * p + 1] : k_eff);
  for (int e = lane; e < max(na, nb); e += 32) {
    if (e < na) {
      const int ja = ra[e];
      atomicOr(&bma[ja >> 5], 1u << (ja & 31));
    }
    if (e < nb) {
      const int jb = rb[e];
      atomicOr(&bmb[jb >> 5], 1u << (jb & 31));
    }
  }
  __syncwarp();
  // class sizes: both, only tile 0, only tile 1
  int n3 = 0, n1 = 0, n2 = 0;
  for (int w = lane; w < nw; w += 32) {
    const uint32_t wa = bma[w], wb = bmb[w];
    n3 += __popc(wa & wb); n1 += __popc(wa & ~wb); n2 += __popc(wb & ~wa);
  }
  n3 = __reduce_add_sync(0xffffffffu, n3);
  n1 = __reduce_add_sync(0xffffffffu, n1);
  n2 = __reduce_add_sync(0xffffffffu, n2);
  int32_t* out = sel_pair + ((int64_t)h * NP + p) * 2 * kcap;
  int base3 = 0, base1 = 0, base2 = 0;                 // entries of each class in the words before this round
  for (int w0 = 0; w0 < nw; w0 += 32) {
    const int w = w0 + lane;
    const uint32_t wa = w < nw ? bma[w] : 0u, wb = w < nw ? bmb[w] : 0u;
    const int c3 = __popc(wa & wb), c1 = __popc(wa & ~wb), c2 = __popc(wb & ~wa);
    int i3 = c3, i1 = c1, i2 = c2;                      // inclusive warp scans
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y3 = __shfl_up_sync(0xffffffffu, i3, o), y1 = __shfl_up_sync(0xffffffffu, i1, o),
                y2 = __shfl_up_sync(0xffffffffu, i2, o);
      if (lane >= o) { i3 += y3; i1 += y1; i2 += y2; }
    }
    int r3 = base3 + i3 - c3, r1 = base1 + i1 - c1, r2 = base2 + i2 - c2;   // rank within the class
    uint32_t u = wa | wb;
    while (u) {
      const int b = __ffs(u) - 1;
      u &= u - 1;
      int gid, phys, nval;
      uf_cand_lookup(v, w * 32 + b, &gid, &phys, &nval);
      const int mask = ((wa >> b) & 1u) | (((wb >> b) & 1u) << 1);
      int pos;
      if (mask == 3)      { pos = r3; ++r3; }
      else if (mask == 1) { pos = n3 + r1 + min(r1, n2); ++r1; }            // a_i at 2i while b_i exists
      else                { pos = n3 + r2 + min(r2 + 1, n1); ++r2; }        // b_i at 2i + 1 while a_i exists
      out[pos] = uf_entry_pack(phys, nval, mask);
    }
    base3 += __shfl_sync(0xffffffffu, i3, 31);
    base1 += __shfl_sync(0xffffffffu, i1, 31);
    base2 += __shfl_sync(0xffffffffu, i2, 31);
  }
  if (lane == 0) pair_cnt[(int64_t)h * NP + p] = n3 + n1 + n2;
}

// the stand-alone form (only when the score kernel runs one query block per CTA and cannot merge pairs itself)
constexpr int kMergeWarps = 4;
__global__ void __launch_bounds__(kMergeWarps * 32)
uf_pair_merge_kernel(UfView v, const int32_t* __restrict__ sel_rank, const int32_t* __restrict__ sel_cnt,
                     int32_t* __restrict__ sel_pair, int32_t* __restrict__ pair_cnt, int nqb, int k_eff, int kcap) {
  extern __shared__ uint32_t bm_raw[];
  const int np_cur = (nqb + 1) / 2;
  const int nw = (v.n_cand + 31) / 32;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int x = blockIdx.x * kMergeWarps + warp;
  if (x >= v.H * np_cur) return;
  uint32_t* bma = bm_raw + (size_t)warp * 2 * nw;
  uf_merge_pair(v, bma, bma + nw, nw, x / np_cur, x % np_cur, nqb, k_eff, kcap, sel_rank, sel_cnt, sel_pair, pair_cnt, lane);
}

}  // namespace

cudaError_t uf_launch_select(uf_ctx* c, const UfView& v, const __nv_bfloat16* q, int64_t tok_stride,
                             int64_t head_stride, int k_eff, int32_t* idx_out, int32_t* cnt_out,
                             bool paper, int out_stride, cudaStream_t s) {
  const int nqb = uf_ceil_div(v.cur_ntok, v.B);
  const int NP = (v.BPC + 1) / 2;
  // usage statistic (NEXT-3): this call counts into the buffer that is NOT current (the previous score kernel zeroed
  // it) and zeroes the current one for the call after it, so no extra launch sits on the hot path.  The host record
  // (which buffer is current, which chunks its counters refer to) is committed only once the score kernel has been
  // enqueued: a call that fails before that leaves the previous selection's statistic intact and the spare buffer zero.
  const int seq = c->usage_seq ^ 1;
  unsigned long long* usage_cur = c->usage + (size_t)seq * UF_MAXC;
  unsigned long long* usage_next = c->usage + (size_t)(seq ^ 1) * UF_MAXC;
  if (k_eff == 0 && !paper) {
    cudaError_t e0 = cudaMemsetAsync(c->usage, 0, 2 * UF_MAXC * sizeof(unsigned long long), s);
    if (e0 != cudaSuccess) return e0;
    c->usage_n = 0;                                    // both buffers are zero: either may be current
    // no candidates (chunk 0, or window 1): counts are zero, nothing to score
    if (cnt_out) {
      cudaError_t e = cudaMemsetAsync(cnt_out, 0, (size_t)v.H * nqb * sizeof(int32_t), s);
      if (e != cudaSuccess) return e;
    }
    return cudaMemsetAsync(c->pair_cnt, 0, (size_t)v.H * NP * sizeof(int32_t), s);
  }
  dim3 gp(nqb, v.H);
  cudaError_t e = cudaSuccess;
#ifndef UF_SCORE_QG_MAX
#define UF_SCORE_QG_MAX 8
#endif
  int qg = UF_SCORE_QG_MAX;
  auto smem_for = [&](int g) { return (size_t)g * v.d * 8 + (size_t)g * v.n_cand * 8; };
  while (qg > 1 && smem_for(qg) > 160 * 1024) qg >>= 1;
  const size_t smem = smem_for(qg);
  if (smem > 200 * 1024) return cudaErrorInvalidConfiguration;     // > ~25k candidates: not supported
  dim3 gs(uf_ceil_div(nqb, qg), v.H);
  const bool want_pairs = (v.B == 128 && v.d == 128);      // the tcgen05 attention kernels walk per-pair union lists
  const bool fuse_merge = want_pairs && qg >= 2;           // built by the score kernel itself
  const bool deep_prefetch = (int64_t)gs.x * gs.y <= 2 * (int64_t)c->sm_count;
#define UF_SCORE_LAUNCH3(DD, QG, PP, PF)                                                                     \
  {                                                                                                          \
    size_t& attr = c->score_smem_attr[(PP ? 1 : 0) + (PF == 16 ? 2 : 0)][DD == 32 ? 0 : DD == 64 ? 1 : 2]    \
                                     [QG == 8 ? 0 : QG == 4 ? 1 : QG == 2 ? 2 : 3];                          \
    if (smem > 48 * 1024 && smem > attr) {          /* raise the limit once, not on every call */             \
      e = cudaFuncSetAttribute(uf_score_topk_kernel<DD, QG, PP, PF>,                                         \
                               cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                      \
      if (e != cudaSuccess) return e;                                                                        \
      attr = smem;                                                                                           \
    }                                                                                                        \
    uf_score_topk_kernel<DD, QG, PP, PF><<<gs, kScoreThreads, smem, s>>>(                                    \
        v, c->qbar, c->kpool, nqb, k_eff, c->sel_q, c->sel_rank, c->kcap, c->sel_cnt, idx_out, cnt_out,      \
        out_stride, usage_cur, fuse_merge ? c->sel_pair : nullptr, c->pair_cnt, usage_next);                 \
  }
  /* few CTAs per SM: latency-bound, prefetch deep (16 loads ahead, 122 registers); many: keep the occupancy */
#define UF_SCORE_LAUNCH2(DD, QG, PP)                                                                         \
  {                                                                                                          \
    if (deep_prefetch) UF_SCORE_LAUNCH3(DD, QG, PP, 16) else UF_SCORE_LAUNCH3(DD, QG, PP, 4)                 \
  }
#define UF_SCORE_LAUNCH(DD, QG)                                                                              \
  {                                                                                                          \
    if (paper) UF_SCORE_LAUNCH2(DD, QG, true) else UF_SCORE_LAUNCH2(DD, QG, false)                           \
  }
#define UF_SELECT_CASE(DD)                                                                                   \
  case DD:                                                                                                   \
    if (!c->skip_pool_q) {               /* pooled Q already written by uf_qkv_rope_append: nothing to pool */ \
      uf_pool_q_kernel<DD><<<gp, kPoolThreads, 0, s>>>(q, tok_stride, head_stride, c->qbar, v.B, v.BPC,      \
                                                       v.cur_ntok, v.til);                                   \
      c->launches += 1;                                                                                      \
    }                                                                                                        \
    if (qg == 8) UF_SCORE_LAUNCH(DD, 8)                                                                      \
    else if (qg == 4) UF_SCORE_LAUNCH(DD, 4)                                                                 \
    else if (qg == 2) UF_SCORE_LAUNCH(DD, 2)                                                                 \
    else UF_SCORE_LAUNCH(DD, 1)                                                                              \
    break;
  switch (v.d) {
    UF_SELECT_CASE(32)
    UF_SELECT_CASE(64)
    UF_SELECT_CASE(128)
    default: return cudaErrorInvalidValue;
  }
#undef UF_SELECT_CASE
#undef UF_SCORE_LAUNCH
#undef UF_SCORE_LAUNCH2
#undef UF_SCORE_LAUNCH3
  c->launches += 1;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  c->usage_seq = seq;
  c->usage_n = v.n_prior;
  for (int i = 0; i < v.n_prior; ++i) c->usage_chunk[i] = v.prior_chunk[i];
  if (want_pairs && !fuse_merge) {
    const int np_cur = (nqb + 1) / 2;
    const size_t msmem = (size_t)kMergeWarps * 2 * uf_ceil_div(v.n_cand, 32) * sizeof(uint32_t);
    uf_pair_merge_kernel<<<uf_ceil_div(v.H * np_cur, kMergeWarps), kMergeWarps * 32, msmem, s>>>(
        v, c->sel_rank, paper ? c->sel_cnt : nullptr, c->sel_pair, c->pair_cnt, nqb, k_eff, c->kcap);
    c->launches += 1;
    e = cudaGetLastError();
  }
  return e;
}
