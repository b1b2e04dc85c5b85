// uf_api.cu — the C ABI of include/uf.h: ctx life cycle, cache bookkeeping (slot map, FIFO window,
// sink), argument checks and kernel dispatch.  No arithmetic of the method runs on the host except
// the integer cache policy (P:136 (iii), BJ configs[3]; readings R-16/R-17 in DESIGN.md).
#include "uf_internal.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <utility>

namespace {

thread_local std::string g_create_err;

int fail(uf_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_err = msg;
  return code;
}
int fail_cuda(uf_ctx* c, cudaError_t e, const char* what) {
  return fail(c, UF_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define UF_CUDA(c, call)                                          \
  do {                                                            \
    cudaError_t e__ = (call);                                     \
    if (e__ != cudaSuccess) return fail_cuda((c), e__, #call);    \
  } while (0)

int n_blocks(const uf_ctx* c, int ntok) { return uf_ceil_div(ntok, c->cfg.block); }

int n_resident(const uf_ctx* c) {
  int n = 0;
  for (int s = 0; s < c->cfg.capacity_chunks; ++s) n += (c->slot_chunk[s] >= 0);
  return n;
}

// Snapshot of the state for the newest chunk (the "current" one).
// paper = true (Eq. 4 mode, R-31/R-32): the candidate list is every block in the causal mask, i.e. the current
// chunk is listed too, as the last "prior".
bool make_view(const uf_ctx* c, UfView* v, bool paper = false) {
  const int C = c->cfg.capacity_chunks;
  int cur = c->next_chunk - 1;
  if (cur < 0) return false;
  memset(v, 0, sizeof(*v));
  v->til = c->til;
  v->H = c->cfg.n_heads; v->d = c->cfg.head_dim; v->B = c->cfg.block;
  v->BPC = c->BPC; v->S = c->cfg.sink_blocks; v->P = c->P;
  v->cur_chunk = cur; v->cur_slot = -1;
  v->sink_ntok = c->sink_ntok;
  const int n_sink_ids = uf_ceil_div(c->sink_ntok, c->cfg.block);   // sink blocks that exist
  v->n_sink_blocks = cur > 0 ? n_sink_ids : 0;
  // resident chunks in ascending id
  int ids[UF_MAXC], slots[UF_MAXC], n = 0;
  for (int s = 0; s < C; ++s)
    if (c->slot_chunk[s] >= 0) { ids[n] = c->slot_chunk[s]; slots[n] = s; ++n; }
  for (int i = 1; i < n; ++i)
    for (int j = i; j > 0 && ids[j - 1] > ids[j]; --j) {
      int t = ids[j]; ids[j] = ids[j - 1]; ids[j - 1] = t;
      t = slots[j]; slots[j] = slots[j - 1]; slots[j - 1] = t;
    }
  int np = 0, pref = 0;
  for (int i = 0; i < n; ++i) {
    if (ids[i] == cur) {
      v->cur_slot = slots[i]; v->cur_ntok = c->slot_ntok[slots[i]];
      if (!paper) continue;
    }
    int nb = n_blocks(c, c->slot_ntok[slots[i]]);
    int first = (ids[i] == 0) ? (n_sink_ids < nb ? n_sink_ids : nb) : 0;   // CAND excludes SINK ids
    v->prior_chunk[np] = ids[i]; v->prior_slot[np] = slots[i];
    v->prior_ntok[np] = c->slot_ntok[slots[i]]; v->prior_first_b[np] = first;
    v->cand_prefix[np] = pref;
    pref += nb - first;
    ++np;
  }
  v->cand_prefix[np] = pref;
  for (int i = np + 1; i <= UF_MAXC; ++i) v->cand_prefix[i] = pref;
  v->n_prior = np; v->n_cand = pref;
  return v->cur_slot >= 0;
}

int topk_budget(const uf_ctx* c, int n_cand, int topk_count, int topk_percent, int* k_eff) {
  int64_t k;
  if (topk_count >= 0) k = topk_count;
  else {
    if (topk_percent < 0 || topk_percent > 100) return UF_ERR_INVALID_ARG;
    k = ((int64_t)topk_percent * n_cand) / 100;
    if (k < c->cfg.k_min) k = c->cfg.k_min;
  }
  if (k > n_cand) k = n_cand;
  *k_eff = (int)k;
  return UF_OK;
}

int check_tensor_args(uf_ctx* c, const void* p, int64_t tok_stride, int64_t head_stride, const char* name) {
  if (!p) return fail(c, UF_ERR_INVALID_ARG, std::string(name) + ": null pointer");
  if (((uintptr_t)p & 15) != 0) return fail(c, UF_ERR_INVALID_ARG, std::string(name) + ": pointer not 16-byte aligned");
  if (tok_stride < c->cfg.head_dim || head_stride < c->cfg.head_dim || (tok_stride % 8) || (head_stride % 8))
    return fail(c, UF_ERR_INVALID_ARG, std::string(name) + ": strides must be >= head_dim and multiples of 8 elements");
  return UF_OK;
}

// Do two [n, H, d] bf16 tensors (element strides ts, hs, 1) share an element?  Exact for the layouts a QKV projection
// leaves behind when both have the same strides and rows / heads do not overlap themselves (slices of [n, 3, H, d] or
// of [n, H, 3, d]: the byte ranges interleave but no element is shared); conservative (byte ranges) otherwise.
bool tensors_overlap(const void* a, int64_t a_ts, int64_t a_hs, const void* b, int64_t b_ts, int64_t b_hs, int n, int H,
                     int d) {
  auto last = [&](int64_t ts, int64_t hs) { return (int64_t)(n - 1) * ts + (int64_t)(H - 1) * hs + d; };
  const intptr_t pa = (intptr_t)a, pb = (intptr_t)b;
  if (pa + 2 * last(a_ts, a_hs) <= pb || pb + 2 * last(b_ts, b_hs) <= pa) return false;      // disjoint byte ranges
  if (a_ts != b_ts || a_hs != b_hs || ((pb - pa) & 1)) return true;
  const int64_t ts = a_ts, hs = a_hs, hspan = (int64_t)(H - 1) * hs + d;
  if (hspan > ts || d > hs) return true;                                                      // self-overlapping layout
  const int64_t delta = (pb - pa) / 2;
  const int64_t in_row = ((delta % ts) + ts) % ts;              // b's row start relative to the row of a it falls in
  for (int64_t x : {in_row, in_row - ts}) {                     // ... and to the next row of a
    if (x >= hspan || -x >= hspan) continue;                    // the two rows' occupied spans do not meet
    if (H == 1) return true;
    const int64_t y = ((x % hs) + hs) % hs;                     // same question one level down: head windows of d
    if (y < d || hs - y < d) return true;
  }
  return false;
}

void clear_host_state(uf_ctx* c) {
  for (int s = 0; s < UF_MAXC; ++s) { c->slot_chunk[s] = -1; c->slot_ntok[s] = 0; }
  c->next_chunk = 0; c->sink_ntok = 0; c->sel_valid = false; c->sel_k = 0; c->sel_ntok = 0;
  c->usage_n = 0; c->qbar_chunk = -1;
}

// Steps shared by uf_kv_append and uf_qkv_rope_append: the integer cache policy on a copy of the slot state, the
// device work (`launch`, given the view of the new state), commit / roll back.
template <typename Launch>
int32_t append_common(uf_ctx* c, int32_t n_tokens, int32_t window_chunks, const char* name, Launch launch) {
  const int C = c->cfg.capacity_chunks;
  if (n_tokens < 1) return fail(c, UF_ERR_INVALID_ARG, std::string(name) + ": n_tokens < 1");
  if (n_tokens > c->cfg.chunk_tokens_max) return fail(c, UF_ERR_CAPACITY, std::string(name) + ": n_tokens > chunk_tokens_max");
  if (window_chunks < 0 || window_chunks > C) return fail(c, UF_ERR_CAPACITY, std::string(name) + ": window_chunks outside 0..capacity_chunks");
  if (c->til.enabled && n_tokens != c->BPC * c->cfg.block)
    return fail(c, UF_ERR_INVALID_ARG, std::string(name) + ": a tiled ctx takes whole chunks in the tiled layout (n_tokens = N_b * block)");
  // --- cache policy (host, integers only), computed on a copy of the slot state: it is committed only after
  // the device work was enqueued, so a failing launch leaves the ctx as it was ---
  const int cid = c->next_chunk;
  const int W = window_chunks == 0 ? C : window_chunks;
  int slot_chunk[UF_MAXC], slot_ntok[UF_MAXC];
  for (int s = 0; s < UF_MAXC; ++s) { slot_chunk[s] = c->slot_chunk[s]; slot_ntok[s] = c->slot_ntok[s]; }
  for (;;) {   // evict ids <= cid - W, oldest first
    int oldest = -1;
    for (int s = 0; s < C; ++s)
      if (slot_chunk[s] >= 0 && (oldest < 0 || slot_chunk[s] < slot_chunk[oldest])) oldest = s;
    if (oldest < 0 || slot_chunk[oldest] > cid - W) break;
    slot_chunk[oldest] = -1; slot_ntok[oldest] = 0;
  }
  int slot = -1;
  for (int s = 0; s < C; ++s) if (slot_chunk[s] < 0) { slot = s; break; }   // lowest free slot
  if (slot < 0) return fail(c, UF_ERR_STATE, std::string(name) + ": no free slot (internal)");
  slot_chunk[slot] = cid; slot_ntok[slot] = n_tokens;
  int sink_ntok = c->sink_ntok;
  if (cid == 0) {
    int ns = c->cfg.sink_blocks * c->cfg.block;
    sink_ntok = ns < n_tokens ? ns : n_tokens;
  }
  struct Saved { int slot_chunk[UF_MAXC], slot_ntok[UF_MAXC], next_chunk, sink_ntok; bool sel_valid; } old;
  for (int s = 0; s < UF_MAXC; ++s) { old.slot_chunk[s] = c->slot_chunk[s]; old.slot_ntok[s] = c->slot_ntok[s]; }
  old.next_chunk = c->next_chunk; old.sink_ntok = c->sink_ntok; old.sel_valid = c->sel_valid;
  auto rollback = [&]() {
    for (int s = 0; s < UF_MAXC; ++s) { c->slot_chunk[s] = old.slot_chunk[s]; c->slot_ntok[s] = old.slot_ntok[s]; }
    c->sink_ntok = old.sink_ntok; c->next_chunk = old.next_chunk; c->sel_valid = old.sel_valid;
  };
  for (int s = 0; s < UF_MAXC; ++s) { c->slot_chunk[s] = slot_chunk[s]; c->slot_ntok[s] = slot_ntok[s]; }
  c->sink_ntok = sink_ntok; c->next_chunk = cid + 1; c->sel_valid = false;
  c->qbar_chunk = -1;                                   // pooled Q of an older chunk is stale now
  if (c->host_only) return UF_OK;
  // --- device ---
  cudaError_t e = cudaSetDevice(c->cfg.device);
  UfView view;
  if (e == cudaSuccess && !make_view(c, &view)) { rollback(); return fail(c, UF_ERR_STATE, std::string(name) + ": inconsistent slot state (internal)"); }
  if (e == cudaSuccess) e = launch(view);
  if (e != cudaSuccess) {
    rollback();                       // the chunk was not written: the ctx still describes the previous state
    return fail_cuda(c, e, name);
  }
  return UF_OK;
}

}  // namespace

extern "C" {

const char* uf_version(void) { return "uf-b200 0.1 (sm_100a)"; }

const char* uf_last_error(const uf_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

int32_t uf_ctx_create(const uf_config* cfg, uf_ctx** out) {
  if (!cfg || !out) return fail(nullptr, UF_ERR_INVALID_ARG, "uf_ctx_create: null argument");
  *out = nullptr;
  if (cfg->n_heads < 1 || (cfg->head_dim != 32 && cfg->head_dim != 64 && cfg->head_dim != 128) ||
      cfg->block < 32 || cfg->block > 128 || (cfg->block % 32) || cfg->chunk_tokens_max < 1 ||
      cfg->capacity_chunks < 1 || cfg->capacity_chunks > UF_MAXC || cfg->sink_blocks < 0 ||
      cfg->sink_blocks > 4 || cfg->k_min < 0)
    return fail(nullptr, UF_ERR_INVALID_ARG, "uf_ctx_create: config out of range (see uf.h)");
  uf_ctx* c = new (std::nothrow) uf_ctx();
  if (!c) return fail(nullptr, UF_ERR_CAPACITY, "uf_ctx_create: out of host memory");
  c->cfg = *cfg;
  c->BPC = uf_ceil_div(cfg->chunk_tokens_max, cfg->block);
  c->P = cfg->sink_blocks + cfg->capacity_chunks * c->BPC;
  c->kcap = cfg->capacity_chunks * c->BPC;     // a row keeps at most every block in the causal mask (paper-mask mode)
  if (c->P >= (1 << 20)) { delete c; return fail(nullptr, UF_ERR_CAPACITY, "uf_ctx_create: too many physical blocks"); }
  clear_host_state(c);
  c->host_only = cfg->device < 0;
  if (c->host_only) { *out = c; return UF_OK; }

  cudaError_t e = cudaSetDevice(cfg->device);
  if (e != cudaSuccess) { int r = fail_cuda(nullptr, e, "cudaSetDevice"); delete c; return r; }
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, cfg->device);
  if (e != cudaSuccess) { int r = fail_cuda(nullptr, e, "cudaGetDeviceProperties"); delete c; return r; }
  if (prop.major != 10) {
    delete c;
    return fail(nullptr, UF_ERR_UNSUPPORTED, "uf_ctx_create: this library is built for sm_100a (B200) only");
  }
  c->sm_count = prop.multiProcessorCount;
  const int64_t H = cfg->n_heads, d = cfg->head_dim, B = cfg->block, P = c->P, BPC = c->BPC;
  const int64_t NP = (BPC + 1) / 2;
  const int64_t cache_bytes = H * P * B * d * 2;
  struct { void** p; int64_t bytes; } allocs[] = {
      {(void**)&c->kc, cache_bytes},
      {(void**)&c->vc, cache_bytes},
      {(void**)&c->kpool, H * d * P * 8},
      {(void**)&c->qbar, H * BPC * d * 8},
      {(void**)&c->sel_q, H * BPC * (int64_t)c->kcap * 4},
      {(void**)&c->sel_rank, H * BPC * (int64_t)c->kcap * 4},
      {(void**)&c->sel_pair, H * NP * 2 * (int64_t)c->kcap * 4},
      {(void**)&c->pair_cnt, H * NP * 4},
      {(void**)&c->sel_cnt, H * BPC * 4},
      {(void**)&c->usage, 2 * UF_MAXC * 8},
      {(void**)&c->panic_item, H * NP * 4},
      {(void**)&c->panic_last, 4},
  };
  for (auto& a : allocs) {
    e = cudaMalloc(a.p, (size_t)a.bytes);
    if (e != cudaSuccess) {
      int r = fail_cuda(nullptr, e, "cudaMalloc");
      uf_ctx_destroy(c);
      return r;
    }
    c->dev_bytes += a.bytes;
  }
  e = cudaMemset(c->kc, 0, (size_t)cache_bytes);
  if (e == cudaSuccess) e = cudaMemset(c->vc, 0, (size_t)cache_bytes);
  if (e == cudaSuccess) e = cudaMemset(c->kpool, 0, (size_t)(H * d * P * 8));
  if (e == cudaSuccess) e = cudaMemset(c->panic_item, 0, (size_t)(H * NP * 4));
  if (e == cudaSuccess) e = cudaMemset(c->panic_last, 0, 4);
  if (e == cudaSuccess) e = cudaMemset(c->usage, 0, 2 * UF_MAXC * 8);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e != cudaSuccess) { int r = fail_cuda(nullptr, e, "cudaMemset"); uf_ctx_destroy(c); return r; }
  if (cfg->block == 128 && cfg->head_dim == 128) {
    int r = uf_sm100_make_cache_maps(c);
    if (r != UF_OK) { g_create_err = c->err; uf_ctx_destroy(c); return r; }
  }
  *out = c;
  return UF_OK;
}

int32_t uf_ctx_destroy(uf_ctx* c) {
  if (!c) return UF_OK;
  if (!c->host_only) {
    cudaSetDevice(c->cfg.device);
    cudaFree(c->kc); cudaFree(c->vc); cudaFree(c->kpool); cudaFree(c->qbar);
    cudaFree(c->sel_q); cudaFree(c->sel_rank); cudaFree(c->sel_pair); cudaFree(c->pair_cnt);
    cudaFree(c->panic_item); cudaFree(c->panic_last); cudaFree(c->sel_cnt); cudaFree(c->usage);
  }
  delete c;
  return UF_OK;
}

int32_t uf_ctx_reset(uf_ctx* c, void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  (void)stream;
  // Host state only.  Nothing on the device has to be cleared: the append kernel rewrites every row (pad rows as
  // zeros) of every block it makes addressable, the sink region and the pooled-K entries included, and a block
  // that is not addressable through the slot map / sink count is never read.
  clear_host_state(c);
  return UF_OK;
}

int32_t uf_kv_append(uf_ctx* c, const void* k, const void* v, int32_t n_tokens,
                     int64_t tok_stride, int64_t head_stride, int32_t window_chunks, void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (!c->host_only) {
    int r = check_tensor_args(c, k, tok_stride, head_stride, "uf_kv_append k");
    if (r) return r;
    r = check_tensor_args(c, v, tok_stride, head_stride, "uf_kv_append v");
    if (r) return r;
  }
  return append_common(c, n_tokens, window_chunks, "uf_kv_append", [&](const UfView& view) {
    return uf_launch_append(c, view, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, tok_stride, head_stride,
                            (cudaStream_t)stream);
  });
}

// NEXT-2 (R-37..R-40): QK-norm + 3-D RoPE + append + pooled K + pooled Q in one pass
int32_t uf_qkv_rope_append(uf_ctx* c, const void* q_in, const void* k_in, const void* v_in, void* q_out,
                           int32_t n_tokens, int64_t in_tok_stride, int64_t in_head_stride, int64_t out_tok_stride,
                           int64_t out_head_stride, const uf_rope_spec* rs, int32_t window_chunks, void* stream) {
  if (!c || !rs) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_qkv_rope_append: host-only ctx has no device path");
  if (c->cfg.head_dim != 128) return fail(c, UF_ERR_UNSUPPORTED, "uf_qkv_rope_append: head_dim must be 128");
  int r = check_tensor_args(c, q_in, in_tok_stride, in_head_stride, "uf_qkv_rope_append q_in");
  if (!r) r = check_tensor_args(c, k_in, in_tok_stride, in_head_stride, "uf_qkv_rope_append k_in");
  if (!r) r = check_tensor_args(c, v_in, in_tok_stride, in_head_stride, "uf_qkv_rope_append v_in");
  if (!r) r = check_tensor_args(c, q_out, out_tok_stride, out_head_stride, "uf_qkv_rope_append q_out");
  if (r) return r;
  if (!rs->cos_tab || !rs->sin_tab || !rs->gq || !rs->gk)
    return fail(c, UF_ERR_INVALID_ARG, "uf_qkv_rope_append: null table / weight pointer");
  if (n_tokens >= 1) {
    // q_out may be q_in itself (same pointer, same strides: a row is staged on chip before it is overwritten, and no
    // other CTA reads it); every other overlap of q_out with an input would let one CTA overwrite rows another CTA
    // has not read yet
    const bool same_strides = out_tok_stride == in_tok_stride && out_head_stride == in_head_stride;
    auto collides = [&](const void* in) {
      return tensors_overlap(q_out, out_tok_stride, out_head_stride, in, in_tok_stride, in_head_stride, n_tokens,
                             c->cfg.n_heads, c->cfg.head_dim);
    };
    if ((!(q_out == q_in && same_strides) && collides(q_in)) || collides(k_in) || collides(v_in))
      return fail(c, UF_ERR_INVALID_ARG, "uf_qkv_rope_append: q_out overlaps an input (only q_out == q_in with equal strides is allowed)");
  }
  if (rs->dim_t < 0 || rs->dim_h < 0 || rs->dim_w < 0 || (rs->dim_t & 1) || (rs->dim_h & 1) || (rs->dim_w & 1) ||
      rs->dim_t + rs->dim_h + rs->dim_w != c->cfg.head_dim)
    return fail(c, UF_ERR_INVALID_ARG, "uf_qkv_rope_append: axis dims must be even and sum to head_dim");
  if (!(rs->eps >= 0.0) || rs->t0 < 0 || rs->max_pos < 1)
    return fail(c, UF_ERR_INVALID_ARG, "uf_qkv_rope_append: bad eps / t0 / max_pos");
  // the largest position any token of this chunk uses must be inside the tables
  int frames, gh, gw;
  if (c->til.enabled) { frames = c->til.F; gh = c->til.Hg; gw = c->til.Wg; }
  else {
    gh = rs->grid_h; gw = rs->grid_w;
    if (gh < 1 || gw < 1) return fail(c, UF_ERR_INVALID_ARG, "uf_qkv_rope_append: grid_h, grid_w must be >= 1");
    frames = uf_ceil_div(n_tokens, gh * gw);
  }
  if (rs->t0 + frames > rs->max_pos || gh > rs->max_pos || gw > rs->max_pos)
    return fail(c, UF_ERR_CAPACITY, "uf_qkv_rope_append: a position exceeds max_pos (the RoPE tables are too short)");
  int32_t st = append_common(c, n_tokens, window_chunks, "uf_qkv_rope_append", [&](const UfView& view) {
    return uf_launch_fused_append(c, view, (const __nv_bfloat16*)q_in, (const __nv_bfloat16*)k_in,
                                  (const __nv_bfloat16*)v_in, (__nv_bfloat16*)q_out, in_tok_stride, in_head_stride,
                                  out_tok_stride, out_head_stride, rs, (cudaStream_t)stream);
  });
  if (st == UF_OK) {
    // the pooled Q of this chunk is already in the ctx: uf_select_blocks(q_out, ...) skips its pooling pass
    c->qbar_chunk = c->next_chunk - 1; c->qbar_ptr = q_out; c->qbar_ts = out_tok_stride; c->qbar_hs = out_head_stride;
  }
  return st;
}

int32_t uf_set_pooled_q_reuse(uf_ctx* c, int32_t on) {
  if (!c) return UF_ERR_INVALID_ARG;
  c->reuse_pooled_q = on != 0;
  return UF_OK;
}

int32_t uf_query_topk(const uf_ctx* c, int32_t topk_count, int32_t topk_percent, int32_t* n_cand, int32_t* k_eff) {
  if (!c) return UF_ERR_INVALID_ARG;
  UfView v;
  if (!make_view(c, &v)) return UF_ERR_STATE;
  int k = 0;
  int r = topk_budget(c, v.n_cand, topk_count, topk_percent, &k);
  if (r) return r;
  if (n_cand) *n_cand = v.n_cand;
  if (k_eff) *k_eff = k;
  return UF_OK;
}

int32_t uf_select_blocks(uf_ctx* c, const void* q, int32_t n_tokens, int64_t tok_stride, int64_t head_stride,
                         int32_t topk_count, int32_t topk_percent, int32_t* idx_out, int32_t* cnt_out,
                         void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_select_blocks: host-only ctx has no device path");
  UfView v;
  if (!make_view(c, &v)) return fail(c, UF_ERR_STATE, "uf_select_blocks: no chunk appended yet");
  if (c->til.enabled) return fail(c, UF_ERR_STATE, "uf_select_blocks: this ctx is tiled (uf_ctx_set_tiling): use uf_select_blocks_paper");
  if (n_tokens != v.cur_ntok) return fail(c, UF_ERR_INVALID_ARG, "uf_select_blocks: n_tokens differs from the last append");
  int r = check_tensor_args(c, q, tok_stride, head_stride, "uf_select_blocks q");
  if (r) return r;
  int k = 0;
  r = topk_budget(c, v.n_cand, topk_count, topk_percent, &k);
  if (r) return fail(c, r, "uf_select_blocks: topk_percent outside 0..100");
  if (k > c->kcap) return fail(c, UF_ERR_CAPACITY, "uf_select_blocks: k exceeds workspace (internal)");
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  c->skip_pool_q = c->reuse_pooled_q && (c->qbar_chunk == v.cur_chunk && c->qbar_ptr == q && c->qbar_ts == tok_stride && c->qbar_hs == head_stride);
  if (!c->skip_pool_q) c->qbar_chunk = -1;      // this call pools q into the ctx's table: the fused call's pooled Q is gone
  cudaError_t e = uf_launch_select(c, v, (const __nv_bfloat16*)q, tok_stride, head_stride, k, idx_out, cnt_out,
                                   false, k, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "uf_select_blocks kernel launch");
  c->sel_valid = true; c->sel_k = k; c->sel_ntok = n_tokens; c->sel_paper = false;
  return UF_OK;
}

// ---- paper-mask mode (readings R-29..R-35) ----------------

int32_t uf_ctx_set_tiling(uf_ctx* c, const uf_tiling* t) {
  if (!c || !t) return UF_ERR_INVALID_ARG;
  if (c->next_chunk != 0) return fail(c, UF_ERR_STATE, "uf_ctx_set_tiling: the cache is not empty (call before the first append or after uf_ctx_reset)");
  if (t->frames < 1 || t->grid_h < 1 || t->grid_w < 1 || t->bt < 1 || t->bh < 1 || t->bw < 1 ||
      t->window < 1 || (t->window % 2) == 0)
    return fail(c, UF_ERR_INVALID_ARG, "uf_ctx_set_tiling: sizes must be >= 1 and the window odd");
  if ((int64_t)t->bt * t->bh * t->bw != c->cfg.block)
    return fail(c, UF_ERR_INVALID_ARG, "uf_ctx_set_tiling: bt * bh * bw must equal the ctx's block size");
  if (c->cfg.sink_blocks != 0)
    return fail(c, UF_ERR_INVALID_ARG, "uf_ctx_set_tiling: the paper's mask has no sink (create the ctx with sink_blocks = 0)");
  UfTiling u;
  u.enabled = 1;
  u.F = t->frames; u.Hg = t->grid_h; u.Wg = t->grid_w; u.bt = t->bt; u.bh = t->bh; u.bw = t->bw;
  u.nbt = uf_ceil_div(u.F, u.bt); u.nbh = uf_ceil_div(u.Hg, u.bh); u.nbw = uf_ceil_div(u.Wg, u.bw);
  u.half = (t->window - 1) / 2;
  if ((int64_t)u.nbt * u.nbh * u.nbw != c->BPC)
    return fail(c, UF_ERR_INVALID_ARG, "uf_ctx_set_tiling: chunk_tokens_max must be N_b * block with N_b = ceil(F/bt) * ceil(Hg/bh) * ceil(Wg/bw)");
  c->til = u;
  c->sel_valid = false;
  return UF_OK;
}

static int paper_budget(const uf_ctx* c, int n_blocks, int topk_count, int rho_permille, int* k_eff) {
  int64_t k;
  if (topk_count >= 0) k = topk_count;
  else {
    if (rho_permille < 0 || rho_permille > 100000) return UF_ERR_INVALID_ARG;
    // repaired Eq. 10 (R-34): tau_k = max(k_min, floor(rho * 0.42 * N_blocks)), integers only
    k = ((int64_t)rho_permille * 420 * n_blocks) / 1000000;
    if (k < c->cfg.k_min) k = c->cfg.k_min;
  }
  if (k > n_blocks) k = n_blocks;
  *k_eff = (int)k;
  return UF_OK;
}

int32_t uf_query_budget_paper(const uf_ctx* c, int32_t topk_count, int32_t rho_permille, int32_t* n_blocks,
                              int32_t* k_eff) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (!c->til.enabled) return UF_ERR_STATE;
  UfView v;
  if (!make_view(c, &v, true)) return UF_ERR_STATE;
  int k = 0;
  int r = paper_budget(c, v.n_cand, topk_count, rho_permille, &k);
  if (r) return r;
  if (n_blocks) *n_blocks = v.n_cand;
  if (k_eff) *k_eff = k;
  return UF_OK;
}

int32_t uf_select_blocks_paper(uf_ctx* c, const void* q, int32_t n_tokens, int64_t tok_stride, int64_t head_stride,
                               int32_t topk_count, int32_t rho_permille, int32_t* idx_out, int32_t idx_stride,
                               int32_t* cnt_out, void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_select_blocks_paper: host-only ctx has no device path");
  if (!c->til.enabled) return fail(c, UF_ERR_STATE, "uf_select_blocks_paper: call uf_ctx_set_tiling first");
  UfView v;
  if (!make_view(c, &v, true)) return fail(c, UF_ERR_STATE, "uf_select_blocks_paper: no chunk appended yet");
  if (n_tokens != v.cur_ntok) return fail(c, UF_ERR_INVALID_ARG, "uf_select_blocks_paper: n_tokens differs from the last append");
  int r = check_tensor_args(c, q, tok_stride, head_stride, "uf_select_blocks_paper q");
  if (r) return r;
  int k = 0;
  r = paper_budget(c, v.n_cand, topk_count, rho_permille, &k);
  if (r) return fail(c, r, "uf_select_blocks_paper: rho_permille outside 0..100000");
  const int max_row = (k + 1 < v.n_cand ? k + 1 : v.n_cand);          // tau_k blocks + the own block
  if (idx_out && idx_stride < max_row)
    return fail(c, UF_ERR_CAPACITY, "uf_select_blocks_paper: idx_stride < min(k + 1, N_blocks)");
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  c->skip_pool_q = c->reuse_pooled_q && (c->qbar_chunk == v.cur_chunk && c->qbar_ptr == q && c->qbar_ts == tok_stride && c->qbar_hs == head_stride);
  if (!c->skip_pool_q) c->qbar_chunk = -1;      // this call pools q into the ctx's table: the fused call's pooled Q is gone
  cudaError_t e = uf_launch_select(c, v, (const __nv_bfloat16*)q, tok_stride, head_stride, k, idx_out, cnt_out,
                                   true, idx_stride, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "uf_select_blocks_paper kernel launch");
  c->sel_valid = true; c->sel_k = k; c->sel_ntok = n_tokens; c->sel_paper = true;
  return UF_OK;
}

static int32_t tile_call(uf_ctx* c, const void* src, void* dst, int64_t src_ts, int64_t src_hs, int64_t dst_ts,
                         int64_t dst_hs, bool untile, void* stream, const char* name) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, std::string(name) + ": host-only ctx has no device path");
  if (!c->til.enabled) return fail(c, UF_ERR_STATE, std::string(name) + ": call uf_ctx_set_tiling first");
  int r = check_tensor_args(c, src, src_ts, src_hs, name);
  if (r) return r;
  r = check_tensor_args(c, dst, dst_ts, dst_hs, name);
  if (r) return r;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaError_t e = uf_launch_tile(c, (const __nv_bfloat16*)src, (__nv_bfloat16*)dst, src_ts, src_hs, dst_ts, dst_hs,
                                 untile, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail_cuda(c, e, name);
  return UF_OK;
}

int32_t uf_tile_tokens(uf_ctx* c, const void* raster, void* tiled, int64_t raster_tok_stride,
                       int64_t raster_head_stride, int64_t tiled_tok_stride, int64_t tiled_head_stride, void* stream) {
  return tile_call(c, raster, tiled, raster_tok_stride, raster_head_stride, tiled_tok_stride, tiled_head_stride, false,
                   stream, "uf_tile_tokens");
}

int32_t uf_untile_tokens(uf_ctx* c, const void* tiled, void* raster, int64_t tiled_tok_stride,
                         int64_t tiled_head_stride, int64_t raster_tok_stride, int64_t raster_head_stride, void* stream) {
  return tile_call(c, tiled, raster, tiled_tok_stride, tiled_head_stride, raster_tok_stride, raster_head_stride, true,
                   stream, "uf_untile_tokens");
}

int32_t uf_sparse_attn_fwd(uf_ctx* c, const void* q, void* o, float* lse, int32_t n_tokens,
                           int64_t tok_stride, int64_t head_stride, float softmax_scale, void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_sparse_attn_fwd: host-only ctx has no device path");
  UfView v;
  if (!make_view(c, &v)) return fail(c, UF_ERR_STATE, "uf_sparse_attn_fwd: no chunk appended yet");
  if (!c->sel_valid) return fail(c, UF_ERR_STATE, "uf_sparse_attn_fwd: uf_select_blocks / uf_select_blocks_paper must run after the last append");
  if (n_tokens != c->sel_ntok) return fail(c, UF_ERR_INVALID_ARG, "uf_sparse_attn_fwd: n_tokens differs from the selection's");
  int r = check_tensor_args(c, q, tok_stride, head_stride, "uf_sparse_attn_fwd q");
  if (r) return r;
  r = check_tensor_args(c, o, tok_stride, head_stride, "uf_sparse_attn_fwd o");
  if (r) return r;
  if (!(softmax_scale >= 0.0f) || std::isinf(softmax_scale)) return fail(c, UF_ERR_INVALID_ARG, "uf_sparse_attn_fwd: bad softmax_scale");
  float scale = softmax_scale == 0.0f ? (float)(1.0 / std::sqrt((double)c->cfg.head_dim)) : softmax_scale;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  const bool fast = (c->cfg.block == 128 && c->cfg.head_dim == 128 && c->attn_impl != 1 && c->tm_ok);
  if (!fast && c->attn_impl != 1)
    return fail(c, UF_ERR_UNSUPPORTED,
                "uf_sparse_attn_fwd: the tcgen05 kernel needs block == 128 and head_dim == 128; other shapes only run "
                "on the (slow) CUDA-core kernel after uf_set_attn_impl(ctx, 1)");
  if (fast) {
    // the exact-max kernel re-reads Q of the items it redoes after the fast kernel stored their O rows
    const int64_t span = ((int64_t)(n_tokens - 1) * tok_stride + (int64_t)(c->cfg.n_heads - 1) * head_stride +
                          c->cfg.head_dim) * 2;
    const uintptr_t qa = (uintptr_t)q, oa = (uintptr_t)o;
    if (qa < oa + (uintptr_t)span && oa < qa + (uintptr_t)span) {
      // the address ranges interleave: fine when q and o are different slices of one fused tensor, i.e. when
      // no (token, head) row of o can touch a row of q.  Offsets in elements, d = row length:
      //   token level: a token's rows span E = (H-1)*head_stride + d elements; disjoint if the offset between
      //                the bases, modulo tok_stride, leaves E free on both sides;
      //   head level:  if tok_stride is a multiple of head_stride, every row of q starts at 0 mod head_stride
      //                and every row of o at delta mod head_stride.
      const int64_t d = c->cfg.head_dim;
      const int64_t delta = (int64_t)(oa > qa ? oa - qa : qa - oa) / 2;
      const int64_t E = (int64_t)(c->cfg.n_heads - 1) * head_stride + d;
      const int64_t rt = delta % tok_stride, rh = delta % head_stride;
      const bool tok_disjoint = rt >= E && tok_stride - rt >= E;
      const bool head_disjoint = (tok_stride % head_stride == 0) && rh >= d && head_stride - rh >= d;
      if (!tok_disjoint && !head_disjoint)
        return fail(c, UF_ERR_INVALID_ARG, "uf_sparse_attn_fwd: o must not overlap q");
    }
  }
  c->last_attn_sm100 = fast;
  if (fast)
    return uf_launch_attn_sm100(c, v, (const __nv_bfloat16*)q, (__nv_bfloat16*)o, lse, tok_stride, head_stride,
                                scale, (cudaStream_t)stream);
  cudaError_t e = uf_launch_attn_generic(c, v, (const __nv_bfloat16*)q, (__nv_bfloat16*)o, lse, tok_stride,
                                         head_stride, scale, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "uf_sparse_attn_fwd kernel launch");
  return UF_OK;
}

// ---- NEXT-3: SR cache window policy (P:136 (iii); reading R-17 + R-36) ----------------------

int32_t uf_get_select_usage(uf_ctx* c, int64_t* kept_per_chunk, int32_t* chunk_ids, int32_t* n_chunks, void* stream) {
  if (!c || !n_chunks) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_get_select_usage: host-only ctx");
  if (!c->sel_valid) return fail(c, UF_ERR_STATE, "uf_get_select_usage: no selection for the newest chunk");
  *n_chunks = c->usage_n;
  if (c->usage_n == 0) return UF_OK;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  unsigned long long host[UF_MAXC];
  UF_CUDA(c, cudaMemcpyAsync(host, c->usage + (size_t)c->usage_seq * UF_MAXC, sizeof(host), cudaMemcpyDeviceToHost,
                             (cudaStream_t)stream));
  UF_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  for (int i = 0; i < c->usage_n; ++i) {
    if (kept_per_chunk) kept_per_chunk[i] = (int64_t)host[i];
    if (chunk_ids) chunk_ids[i] = c->usage_chunk[i];
  }
  return UF_OK;
}

int32_t uf_next_window(uf_ctx* c, const uf_window_policy* p, int32_t* window_chunks, void* stream) {
  if (!c || !p || !window_chunks) return UF_ERR_INVALID_ARG;
  const int C = c->cfg.capacity_chunks;
  auto clampW = [&](int64_t w) { return (int32_t)(w < 1 ? 1 : (w > C ? C : w)); };
  const int next = c->next_chunk;                       // id of the chunk the window is for
  switch (p->kind) {
    case UF_WIN_FIXED:
      *window_chunks = C;
      return UF_OK;
    case UF_WIN_POSITION:
      if (p->warm_chunks < 0 || p->compact_window < 1) return fail(c, UF_ERR_INVALID_ARG, "uf_next_window: bad position policy");
      *window_chunks = next < p->warm_chunks ? C : clampW(p->compact_window);
      return UF_OK;
    case UF_WIN_MEMORY: {
      if (p->budget_bytes < 0) return fail(c, UF_ERR_INVALID_ARG, "uf_next_window: negative budget");
      const int64_t per_chunk = 2ll * c->cfg.n_heads * c->BPC * c->cfg.block * c->cfg.head_dim * 2;   // K + V slot
      *window_chunks = clampW(p->budget_bytes / per_chunk);
      return UF_OK;
    }
    case UF_WIN_CONTENT: {
      if (p->compact_window < 1 || p->min_share_permille < 0 || p->min_share_permille > 1000)
        return fail(c, UF_ERR_INVALID_ARG, "uf_next_window: bad content policy");
      const int R = n_resident(c);
      int T = clampW(R + 1);                            // resident chunks after the next append under plain FIFO
      *window_chunks = T;
      if (c->host_only || !c->sel_valid || c->usage_n == 0) return UF_OK;      // nothing measured yet: keep everything
      int64_t kept[UF_MAXC];
      int32_t ids[UF_MAXC], n = 0;
      int r = uf_get_select_usage(c, kept, ids, &n, stream);
      if (r) return r;
      int64_t total = 0;
      for (int i = 0; i < n; ++i) total += kept[i];
      if (total == 0) return UF_OK;
      // listed chunks ascend in id.  The FIFO victim (if the cache is full) goes anyway; after it, keep evicting the
      // oldest survivor while it holds less than min_share_permille of the kept blocks.  The newest chunk (listed
      // in paper-mask mode only) is never a victim.
      int j = (R + 1 > C) ? 1 : 0;
      while (j < n && ids[j] != c->next_chunk - 1 && T > p->compact_window &&
             kept[j] * 1000 / total < p->min_share_permille) {
        --T; ++j;
      }
      *window_chunks = clampW(T);
      return UF_OK;
    }
    default:
      return fail(c, UF_ERR_INVALID_ARG, "uf_next_window: unknown policy kind");
  }
}

int32_t uf_set_attn_impl(uf_ctx* c, int32_t impl) {
  if (!c || impl < 0 || impl > 2) return UF_ERR_INVALID_ARG;
  c->attn_impl = impl;
  return UF_OK;
}

int32_t uf_get_slot_map(const uf_ctx* c, int32_t* slot_chunk, int32_t* n_res, int32_t* newest) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (slot_chunk) for (int s = 0; s < c->cfg.capacity_chunks; ++s) slot_chunk[s] = c->slot_chunk[s];
  if (n_res) *n_res = n_resident(c);
  if (newest) *newest = c->next_chunk - 1;
  return UF_OK;
}

static int resolve_phys(uf_ctx* c, int32_t g, int* phys) {
  if (g < 0) {
    int s = -g - 1;
    if (s >= uf_ceil_div(c->sink_ntok, c->cfg.block)) return fail(c, UF_ERR_INVALID_ARG, "sink block does not exist");
    *phys = s;
    return UF_OK;
  }
  int cid = g / c->BPC, b = g % c->BPC;
  for (int s = 0; s < c->cfg.capacity_chunks; ++s)
    if (c->slot_chunk[s] == cid) {
      if (b >= n_blocks(c, c->slot_ntok[s])) return fail(c, UF_ERR_INVALID_ARG, "block index past the chunk's last block");
      *phys = c->cfg.sink_blocks + s * c->BPC + b;
      return UF_OK;
    }
  return fail(c, UF_ERR_STATE, "chunk of the requested block is not resident");
}

int32_t uf_get_cache_block(uf_ctx* c, int32_t g, int32_t head, void* k_out, void* v_out, void* stream) {
  if (!c) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_get_cache_block: host-only ctx");
  if (head < 0 || head >= c->cfg.n_heads) return fail(c, UF_ERR_INVALID_ARG, "uf_get_cache_block: bad head");
  int phys = 0;
  int r = resolve_phys(c, g, &phys);
  if (r) return r;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  const int64_t B = c->cfg.block, d = c->cfg.head_dim;
  const int64_t off = ((int64_t)head * c->P + phys) * B * d;
  cudaStream_t s = (cudaStream_t)stream;
  if (k_out) UF_CUDA(c, cudaMemcpyAsync(k_out, c->kc + off, (size_t)(B * d * 2), cudaMemcpyDeviceToHost, s));
  if (v_out) UF_CUDA(c, cudaMemcpyAsync(v_out, c->vc + off, (size_t)(B * d * 2), cudaMemcpyDeviceToHost, s));
  UF_CUDA(c, cudaStreamSynchronize(s));
  return UF_OK;
}

int32_t uf_get_pooled_k(uf_ctx* c, int32_t g, int32_t head, double* out, void* stream) {
  if (!c || !out) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_get_pooled_k: host-only ctx");
  if (head < 0 || head >= c->cfg.n_heads) return fail(c, UF_ERR_INVALID_ARG, "uf_get_pooled_k: bad head");
  int phys = 0;
  int r = resolve_phys(c, g, &phys);
  if (r) return r;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t d = c->cfg.head_dim;
  // kpool is [H][d][P]: a strided gather of d doubles
  UF_CUDA(c, cudaMemcpy2DAsync(out, 8, c->kpool + ((int64_t)head * d) * c->P + phys, (size_t)c->P * 8, 8, (size_t)d,
                               cudaMemcpyDeviceToHost, s));
  UF_CUDA(c, cudaStreamSynchronize(s));
  return UF_OK;
}

int64_t uf_ctx_device_bytes(const uf_ctx* c) { return c ? c->dev_bytes : 0; }
int64_t uf_ctx_launch_count(const uf_ctx* c) { return c ? c->launches : 0; }

int32_t uf_attn_redone_items(uf_ctx* c, int32_t* n_items, void* stream) {
  if (!c || !n_items) return UF_ERR_INVALID_ARG;
  if (c->host_only) return fail(c, UF_ERR_STATE, "uf_attn_redone_items: host-only ctx");
  *n_items = 0;
  if (c->attn_seq == 0 || !c->last_attn_sm100) return UF_OK;
  UF_CUDA(c, cudaSetDevice(c->cfg.device));
  UF_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  const size_t n = (size_t)c->cfg.n_heads * ((c->BPC + 1) / 2);
  int32_t* host = new (std::nothrow) int32_t[n];
  if (!host) return fail(c, UF_ERR_CAPACITY, "uf_attn_redone_items: out of host memory");
  cudaError_t e = cudaMemcpy(host, c->panic_item, n * sizeof(int32_t), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) { delete[] host; return fail_cuda(c, e, "cudaMemcpy(panic_item)"); }
  int cnt = 0;
  for (size_t i = 0; i < n; ++i) cnt += (host[i] == c->attn_seq);
  delete[] host;
  *n_items = cnt;
  return UF_OK;
}

}  // extern "C"
