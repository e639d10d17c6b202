// rbq_api.cu -- host side of the C ABI declared in include/rbq.h: argument checks, workspace
// carve-up, stream/event ordering of the lazy flush.  Every entry point only enqueues kernels.
#include <new>
#include <stdlib.h>
#include <string.h>

#include "rbq_common.cuh"

namespace {

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

void layout_workspace(rbq_ctx* c) {
  const rbq_config& g = c->cfg;
  const size_t B = g.batch, Hq = g.n_q_heads, Hkv = g.n_kv_heads, L = g.max_tokens;
  const size_t rows = B * Hq;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  c->off_qconst = take(B * Hkv * sizeof(RbqQConst));
  c->off_scores = take(rows * L * sizeof(float));
  c->off_selbits = take(rows * (size_t)rbq_words_per_row(c) * sizeof(uint32_t));
  c->off_selcnt = take(rows * sizeof(int32_t));
  c->off_ulist = take(B * Hkv * L * sizeof(uint32_t));
  c->off_ucount = take(B * Hkv * sizeof(int32_t));
  c->off_gdone = take(B * Hkv * sizeof(int32_t));
  c->off_gnext = take(B * Hkv * sizeof(int32_t));
  c->off_rho = take(B * Hkv * sizeof(float));
  c->off_uexact = take(B * Hkv * sizeof(int32_t));
  c->off_rowmax = take(rows * sizeof(uint32_t));
  c->off_part = take(rbq_attention_part_bytes(c));
  const size_t D = g.head_dim;
  c->off_stage_q = take(rows * D * sizeof(float));
  c->off_stage_out = take(rows * D * sizeof(float));
  c->off_centroid = take(B * Hkv * 64 * D * sizeof(double));
  c->off_flags = take(sizeof(uint32_t));
  c->total_bytes = off;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int check_kv(rbq_ctx* ctx, const rbq_kv* kv) {
  if (!kv || !kv->k || !kv->v) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_kv: null pointer");
  if (kv->stride_t < ctx->cfg.head_dim || (kv->stride_t % 8) || (kv->stride_h % 8) || (kv->stride_b % 8))
    RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_kv: strides must be multiples of 8 elements and stride_t >= head_dim");
  if (!aligned16(kv->k) || !aligned16(kv->v)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_kv: k/v must be 16-byte aligned");
  return RBQ_OK;
}

int check_idx(rbq_ctx* ctx, const rbq_index* idx, bool need_codes) {
  if (!idx || !idx->c_k || !idx->n_indexed || !idx->n_total) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_index: null pointer");
  if (need_codes && (!idx->codes || !idx->f_scale)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_index: codes/f_scale null");
  if (need_codes && (!aligned16(idx->codes) || !aligned16(idx->f_scale)))
    RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_index: codes/f_scale must be 16-byte aligned");
  if ((idx->c_q != nullptr) != (idx->f_bias != nullptr))
    RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_index: f_bias must be non-NULL exactly when c_q is");
  return RBQ_OK;
}

int need_ws(rbq_ctx* ctx) {
  if (!ctx->ws || ctx->ws_bytes < ctx->total_bytes)
    RBQ_FAIL(ctx, RBQ_ERR_WORKSPACE, "workspace missing or smaller than rbq_workspace_bytes (%zu)", ctx->total_bytes);
  return RBQ_OK;
}

RbqKV dev_kv(const rbq_kv* kv) { return RbqKV{kv->k, kv->v, (long long)kv->stride_b, (long long)kv->stride_h, (long long)kv->stride_t}; }

template <typename T>
T* ws_ptr(rbq_ctx* ctx, size_t off) { return reinterpret_cast<T*>(static_cast<char*>(ctx->ws) + off); }

}  // namespace

#define RBQ_TRY(expr) do { int rc_ = (expr); if (rc_ != RBQ_OK) return rc_; } while (0)
#define RBQ_CTX(ctx) do { if (!(ctx)) return RBQ_ERR_INVALID_ARG; (ctx)->err[0] = 0; } while (0)

extern "C" {

int rbq_create(const rbq_config* cfg, rbq_ctx** out) {
  if (!cfg || !out) return RBQ_ERR_INVALID_ARG;
  *out = nullptr;
  if (cfg->batch <= 0 || cfg->n_q_heads <= 0 || cfg->n_kv_heads <= 0 || cfg->max_tokens <= 0) return RBQ_ERR_INVALID_ARG;
  if (cfg->n_q_heads % cfg->n_kv_heads) return RBQ_ERR_INVALID_ARG;
  if (cfg->head_dim != 64 && cfg->head_dim != 128 && cfg->head_dim != 256)
    return (cfg->head_dim > 0 && cfg->head_dim % 32 == 0) ? RBQ_ERR_UNSUPPORTED : RBQ_ERR_INVALID_ARG;
  const int G = cfg->n_q_heads / cfg->n_kv_heads;
  if (G != 1 && G != 2 && G != 4) return RBQ_ERR_UNSUPPORTED;
  if (cfg->max_tokens % 4) return RBQ_ERR_INVALID_ARG;
  if (cfg->flush_tokens < 0) return RBQ_ERR_INVALID_ARG;
  for (int d : {cfg->kv_dtype, cfg->q_dtype, cfg->out_dtype})
    if (d != RBQ_F32 && d != RBQ_BF16) return RBQ_ERR_INVALID_ARG;
  if (cfg->rot_kind != RBQ_ROT_DENSE && cfg->rot_kind != RBQ_ROT_WH) return RBQ_ERR_INVALID_ARG;
  if (cfg->factor_dtype != RBQ_F32 && cfg->factor_dtype != RBQ_F16) return RBQ_ERR_INVALID_ARG;
  // tensor-core rotation: built for bf16 K/V (either rotation kind: the WH rotation runs as its dense matrix)
  if (cfg->enc_mode == RBQ_ENC_FAST && (cfg->kv_dtype != RBQ_BF16 || cfg->head_dim != 128)) return RBQ_ERR_UNSUPPORTED;
  if (cfg->enc_mode != RBQ_ENC_EXACT && cfg->enc_mode != RBQ_ENC_FAST) return RBQ_ERR_INVALID_ARG;
  if (!cfg->rot || !(cfg->sm_scale >= 0.0f)) return RBQ_ERR_INVALID_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return RBQ_ERR_CUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return RBQ_ERR_CUDA;
  rbq_ctx* c = new (std::nothrow) rbq_ctx();
  if (!c) return RBQ_ERR_INVALID_ARG;
  memset(c, 0, sizeof(*c));
  c->cfg = *cfg;
  c->G = G;
  c->sm_scale = cfg->sm_scale > 0.0f ? cfg->sm_scale : (float)(1.0 / sqrt((double)cfg->head_dim));
  c->sm_count = sms;
  if (cudaEventCreateWithFlags(&c->ev_copy, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_flush, cudaEventDisableTiming) != cudaSuccess) {
    delete c;
    return RBQ_ERR_CUDA;
  }
  layout_workspace(c);
  // S7 (bf16, head_dim <= 128) straight from the bitmaps; RBQ_GATHER_PLAN=1 in the environment: through the plan kernel and
  // union lists instead (static partition: bit-reproducible accumulation order, ~7 us slower at config 2)
  { const char* e = getenv("RBQ_GATHER_PLAN"); c->gather_via_plan = (e && e[0] == '1') ? 1 : 0; }
  if (rbq_topp_init(c) != RBQ_OK) {
    cudaEventDestroy(c->ev_copy);
    cudaEventDestroy(c->ev_flush);
    delete c;
    return RBQ_ERR_CUDA;
  }
  *out = c;
  return RBQ_OK;
}

int rbq_destroy(rbq_ctx* ctx) {
  if (!ctx) return RBQ_ERR_INVALID_ARG;
  cudaEventDestroy(ctx->ev_copy);
  cudaEventDestroy(ctx->ev_flush);
  if (ctx->host_graph_state == 1) cudaGraphExecDestroy(ctx->host_graph);
  if (ctx->prof_ev) {
    for (int i = 0; i < RBQ_PROFILE_MAX_STEPS * (RBQ_N_STAGES + 1); ++i) cudaEventDestroy(ctx->prof_ev[i]);
    delete[] ctx->prof_ev;
  }
  delete ctx;
  return RBQ_OK;
}

int rbq_workspace_bytes(const rbq_ctx* ctx, size_t* bytes) {
  if (!ctx || !bytes) return RBQ_ERR_INVALID_ARG;
  *bytes = ctx->total_bytes;
  return RBQ_OK;
}

int rbq_set_workspace(rbq_ctx* ctx, void* dev, size_t bytes) {
  RBQ_CTX(ctx);
  if (!dev || (reinterpret_cast<uintptr_t>(dev) & 255u)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
  if (bytes < ctx->total_bytes) RBQ_FAIL(ctx, RBQ_ERR_WORKSPACE, "workspace too small: %zu < %zu", bytes, ctx->total_bytes);
  // a captured host-step graph holds pointers into the old workspace: drop it
  if (ctx->host_graph_state == 1) { cudaGraphExecDestroy(ctx->host_graph); ctx->host_graph = nullptr; }
  if (ctx->host_graph_state > 0) ctx->host_graph_state = 0;
  ctx->ws = dev;
  ctx->ws_bytes = bytes;
  // the sticky status word starts clear (setup call: a blocking 4-byte memset on the legacy stream)
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_flags, 0, sizeof(uint32_t)));
  // row-maximum keys: zero between decode steps (S5 accumulates with atomicMax, S6 clears after reading)
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_rowmax, 0, (size_t)ctx->cfg.batch * ctx->cfg.n_q_heads * sizeof(uint32_t)));
  // per-group arrival and chunk counters of S7: zero between steps (the last CTA to finish a group clears them)
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_gdone, 0, (size_t)ctx->cfg.batch * ctx->cfg.n_kv_heads * sizeof(int32_t)));
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_gnext, 0, (size_t)ctx->cfg.batch * ctx->cfg.n_kv_heads * sizeof(int32_t)));
  // union-size history of S7 (rho = 0: none yet) and its per-step row counters
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_rho, 0, (size_t)ctx->cfg.batch * ctx->cfg.n_kv_heads * sizeof(float)));
  RBQ_CUDA_OK(ctx, cudaMemset(static_cast<char*>(dev) + ctx->off_uexact, 0, (size_t)ctx->cfg.batch * ctx->cfg.n_kv_heads * sizeof(int32_t)));
  return RBQ_OK;
}

int rbq_status_flags(rbq_ctx* ctx, uint32_t* flags_host, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(need_ws(ctx));
  if (!flags_host) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "flags_host null");
  cudaStream_t s = (cudaStream_t)stream;
  RBQ_CUDA_OK(ctx, cudaMemcpyAsync(flags_host, ws_ptr<char>(ctx, ctx->off_flags), sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
  RBQ_CUDA_OK(ctx, cudaStreamSynchronize(s));
  return RBQ_OK;
}

const char* rbq_last_error(const rbq_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int64_t rbq_launch_count(const rbq_ctx* ctx) { return ctx ? ctx->launches : 0; }

int rbq_encode_keys(rbq_ctx* ctx, const rbq_kv* cache, const int32_t* seq_lens, uint32_t flags, rbq_index* idx, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_kv(ctx, cache));
  RBQ_TRY(check_idx(ctx, idx, true));
  RBQ_TRY(need_ws(ctx));
  if (!seq_lens) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "seq_lens null");
  cudaStream_t s = (cudaStream_t)stream;
  const RbqKV kv = dev_kv(cache);
  if (!(flags & RBQ_CK_GIVEN)) RBQ_TRY(rbq_launch_centroid(ctx, kv, seq_lens, idx->c_k, s));
  RBQ_TRY(rbq_launch_encode(ctx, kv, nullptr, seq_lens, 0, ctx->cfg.max_tokens, idx, s));
  RBQ_TRY(rbq_launch_set_counts(ctx, seq_lens, idx->n_indexed, idx->n_total, s));
  ctx->pending = 0;
  ctx->in_flight = 0;
  return RBQ_OK;
}

int rbq_append_tokens(rbq_ctx* ctx, const void* k_new, const void* v_new, int32_t n_new, rbq_kv* cache, rbq_index* idx,
                      void* stream, void* side_stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_kv(ctx, cache));
  RBQ_TRY(check_idx(ctx, idx, true));
  RBQ_TRY(need_ws(ctx));
  if (n_new < 0 || (n_new > 0 && (!k_new || !v_new))) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "k_new/v_new null or n_new < 0");
  if (n_new > 0 && (!aligned16(k_new) || !aligned16(v_new))) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "k_new/v_new must be 16-byte aligned");
  cudaStream_t s = (cudaStream_t)stream, side = (cudaStream_t)side_stream;
  const RbqKV kv = dev_kv(cache);
  int commit = 0;
  if (ctx->in_flight > 0) {                       // (1) commit the flush enqueued by an earlier call
    if (side != s) RBQ_CUDA_OK(ctx, cudaStreamWaitEvent(s, ctx->ev_flush, 0));
    commit = ctx->in_flight;
    ctx->pending -= commit;
    ctx->in_flight = 0;
  }
  RBQ_TRY(rbq_launch_append_copy(ctx, k_new, v_new, n_new, kv, idx->n_indexed, idx->n_total, commit, s));   // (2)
  ctx->pending += n_new;
  const int W = ctx->cfg.flush_tokens;
  if (W > 0 && ctx->pending >= W) {               // (3) batched encode of the oldest whole windows
    const int nf = ctx->pending / W * W;
    if (side != s) {
      RBQ_CUDA_OK(ctx, cudaEventRecord(ctx->ev_copy, s));
      RBQ_CUDA_OK(ctx, cudaStreamWaitEvent(side, ctx->ev_copy, 0));
    }
    RBQ_TRY(rbq_launch_encode(ctx, kv, idx->n_indexed, nullptr, nf, nf, idx, side));
    if (side != s) RBQ_CUDA_OK(ctx, cudaEventRecord(ctx->ev_flush, side));
    ctx->in_flight = nf;
  }
  return RBQ_OK;
}

int rbq_query_quantize(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu, float* qparams, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, false));
  RBQ_TRY(need_ws(ctx));
  if (!q) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q null");
  return rbq_launch_query(ctx, q, idx, qu, qparams, nullptr, false, (cudaStream_t)stream);
}

int rbq_int4_dot_binary(rbq_ctx* ctx, const void* q, const rbq_index* idx, int32_t* dot, int32_t* pop, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, true));
  RBQ_TRY(need_ws(ctx));
  if (!q || !dot || !pop) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q/dot/pop null");
  RBQ_TRY(rbq_launch_query(ctx, q, idx, nullptr, nullptr, nullptr, false, (cudaStream_t)stream));
  return rbq_launch_estimate(ctx, idx, nullptr, dot, pop, nullptr, (cudaStream_t)stream);
}

int rbq_estimate_scores(rbq_ctx* ctx, const void* q, const rbq_index* idx, float* scores, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, true));
  RBQ_TRY(need_ws(ctx));
  if (!q || !scores) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q/scores null");
  if (!aligned16(scores)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores must be 16-byte aligned");
  RBQ_TRY(rbq_launch_query(ctx, q, idx, nullptr, nullptr, nullptr, false, (cudaStream_t)stream));
  return rbq_launch_estimate(ctx, idx, scores, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int rbq_topp_select(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p, int32_t* sel_idx, int32_t* sel_cnt,
                    void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, false));
  RBQ_TRY(need_ws(ctx));
  if (!scores || !sel_idx || !sel_cnt) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores/sel_idx/sel_cnt null");
  if (!aligned16(scores)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores must be 16-byte aligned");
  if (!(p > 0.0f)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "p must be > 0");
  return rbq_launch_topp(ctx, scores, nullptr, idx->n_indexed, p, ws_ptr<uint32_t>(ctx, ctx->off_selbits), sel_idx, sel_cnt,
                         (cudaStream_t)stream);
}

int rbq_topp_select_static(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p, int32_t* sel_idx, int32_t* sel_cnt,
                           void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, false));                          // no need_ws: this entry point uses no workspace
  if (!scores || !sel_idx || !sel_cnt) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores/sel_idx/sel_cnt null");
  if (!aligned16(scores)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores must be 16-byte aligned");
  if (!(p > 0.0f)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "p must be > 0");
  return rbq_launch_topp_static(ctx, scores, idx->n_indexed, p, sel_idx, sel_cnt, (cudaStream_t)stream);
}

int rbq_topp_select_alg3(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p, int32_t* sel_idx, int32_t* sel_cnt,
                         int32_t* iters, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_idx(ctx, idx, false));
  if (!scores || !sel_idx || !sel_cnt) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "scores/sel_idx/sel_cnt null");
  if (!(p > 0.0f)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "p must be > 0");
  return rbq_launch_topp_alg3(ctx, scores, idx->n_indexed, p, sel_idx, sel_cnt, iters, (cudaStream_t)stream);
}

int rbq_sparse_attention(rbq_ctx* ctx, const void* q, const rbq_kv* cache, const rbq_index* idx, const int32_t* sel_idx,
                         const int32_t* sel_cnt, void* out, float* lse, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_kv(ctx, cache));
  RBQ_TRY(check_idx(ctx, idx, false));
  RBQ_TRY(need_ws(ctx));
  if (!q || !sel_idx || !sel_cnt || !out) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q/sel_idx/sel_cnt/out null");
  uint32_t* bits = ws_ptr<uint32_t>(ctx, ctx->off_selbits);
  RBQ_TRY(rbq_launch_bits_from_lists(ctx, idx, sel_idx, sel_cnt, bits, (cudaStream_t)stream));
  return rbq_launch_attention(ctx, q, dev_kv(cache), idx, bits, sel_cnt, out, lse, (cudaStream_t)stream);
}

// q_copy != NULL: q is readable by the device but far away (mapped host memory): S3 reads it once and leaves a device copy
// in q_copy, which S7 (every warp of the gather reads q) uses instead.
static int decode_step_impl(rbq_ctx* ctx, const void* q, void* q_copy, const rbq_kv* cache, const rbq_index* idx, float p, void* out,
                            int32_t* sel_idx, int32_t* sel_cnt, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(check_kv(ctx, cache));
  RBQ_TRY(check_idx(ctx, idx, true));
  RBQ_TRY(need_ws(ctx));
  if (!q || !out) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q/out null");
  if (!(p > 0.0f)) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "p must be > 0");
  cudaStream_t s = (cudaStream_t)stream;
  float* scores = ws_ptr<float>(ctx, ctx->off_scores);
  uint32_t* bits = ws_ptr<uint32_t>(ctx, ctx->off_selbits);
  int32_t* sn = sel_cnt ? sel_cnt : ws_ptr<int32_t>(ctx, ctx->off_selcnt);
  cudaEvent_t* ev = nullptr;                       // stage timing events of this step, if profiling
  if (ctx->prof_on && ctx->prof_steps < RBQ_PROFILE_MAX_STEPS) ev = ctx->prof_ev + (size_t)ctx->prof_steps++ * (RBQ_N_STAGES + 1);
  ctx->stage_ev = ev;
  uint32_t* rowmax = ws_ptr<uint32_t>(ctx, ctx->off_rowmax);   // zero between steps: S6 clears each key once it has read it
  if (ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ev[0], s));
  RBQ_TRY(rbq_launch_query(ctx, q, idx, nullptr, nullptr, q_copy, /*pdl=*/q_copy == nullptr && ev == nullptr, s));
  if (ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ev[1], s));
  RBQ_TRY(rbq_launch_estimate(ctx, idx, scores, nullptr, nullptr, rowmax, s));
  if (ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ev[2], s));
  RBQ_TRY(rbq_launch_topp(ctx, scores, rowmax, idx->n_indexed, p, bits, sel_idx, sn, s));
  if (ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ev[3], s));
  const int rc = rbq_launch_attention(ctx, q_copy ? q_copy : q, dev_kv(cache), idx, bits, sn, out, nullptr, s);   // records ev[4] after the plan
  ctx->stage_ev = nullptr;
  if (rc == RBQ_OK && ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ev[RBQ_N_STAGES], s));
  return rc;
}

int rbq_decode_step(rbq_ctx* ctx, const void* q, const rbq_kv* cache, const rbq_index* idx, float p, void* out,
                    int32_t* sel_idx, int32_t* sel_cnt, void* stream) {
  return decode_step_impl(ctx, q, nullptr, cache, idx, p, out, sel_idx, sel_cnt, stream);
}

int rbq_profile_enable(rbq_ctx* ctx, int enable) {
  RBQ_CTX(ctx);
  if (enable && !ctx->prof_ev) {
    const int n = RBQ_PROFILE_MAX_STEPS * (RBQ_N_STAGES + 1);
    ctx->prof_ev = new (std::nothrow) cudaEvent_t[n];
    if (!ctx->prof_ev) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "out of host memory");
    for (int i = 0; i < n; ++i) RBQ_CUDA_OK(ctx, cudaEventCreate(&ctx->prof_ev[i]));
  }
  ctx->prof_on = enable ? 1 : 0;
  ctx->prof_steps = 0;
  return RBQ_OK;
}

int rbq_profile_read(rbq_ctx* ctx, float* ms_host, int32_t* n_steps_host) {
  RBQ_CTX(ctx);
  if (!ms_host || !n_steps_host) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "ms_host/n_steps_host null");
  for (int k = 0; k < RBQ_N_STAGES; ++k) ms_host[k] = 0.0f;
  *n_steps_host = ctx->prof_steps;
  for (int i = 0; i < ctx->prof_steps; ++i) {
    cudaEvent_t* ev = ctx->prof_ev + (size_t)i * (RBQ_N_STAGES + 1);
    RBQ_CUDA_OK(ctx, cudaEventSynchronize(ev[RBQ_N_STAGES]));
    const bool no_plan = rbq_attention_from_bits(ctx);          // S7 straight from the bitmaps: event 4 is not recorded
    for (int k = 0; k < RBQ_N_STAGES; ++k) {
      if (no_plan && k == 3) continue;                          // plan stage: no launch, 0 ms
      float ms = 0.0f;
      RBQ_CUDA_OK(ctx, cudaEventElapsedTime(&ms, ev[(no_plan && k == 4) ? 3 : k], ev[k + 1]));
      ms_host[k] += ms;
    }
  }
  ctx->prof_steps = 0;
  return RBQ_OK;
}

int rbq_probe_dump(rbq_ctx* ctx, int kernel, uint64_t* out_host) {
  RBQ_CTX(ctx);
  if (!out_host) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "out_host null");
  unsigned long long* o = reinterpret_cast<unsigned long long*>(out_host);
  switch (kernel) {
    case RBQ_PROBE_ESTIMATE: return rbq_probe_copy_estimate(o);
    case RBQ_PROBE_TOPP: return rbq_probe_copy_topp(o);
    case RBQ_PROBE_GATHER: return rbq_probe_copy_gather(o);
    case RBQ_PROBE_PLAN: return rbq_probe_copy_plan(o);
    case RBQ_PROBE_QUERY: return rbq_probe_copy_query(o);
    default: RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "unknown probe kernel %d", kernel);
  }
}

int rbq_decode_step_host(rbq_ctx* ctx, const void* q_host, const rbq_kv* cache, const rbq_index* idx, float p,
                         void* out_host, void* stream) {
  RBQ_CTX(ctx);
  RBQ_TRY(need_ws(ctx));
  if (!q_host || !out_host || !cache || !idx) RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "q_host/out_host/cache/idx null");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t rows = (size_t)ctx->cfg.batch * ctx->cfg.n_q_heads;
  const size_t qb = rows * ctx->cfg.head_dim * (ctx->cfg.q_dtype == RBQ_BF16 ? 2 : 4);
  const size_t ob = rows * ctx->cfg.head_dim * (ctx->cfg.out_dtype == RBQ_BF16 ? 2 : 4);
  void* dq = ws_ptr<char>(ctx, ctx->off_stage_q);
  void* dout = ws_ptr<char>(ctx, ctx->off_stage_out);
  // out_host in pinned (page-locked, mapped) memory: the merge of S7 stores the result straight into it over PCIe and the
  // device-to-host copy disappears; pageable memory goes through the staging buffer.  q is always staged: every warp of the
  // gather reads it.
  auto mapped = [&](const void* h) -> void* {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer && aligned16(at.devicePointer))
      return at.devicePointer;
    cudaGetLastError();
    return nullptr;
  };
  void* out_mapped = nullptr;
  const void* q_mapped = nullptr;                              // S3 reads q over PCIe and leaves the device copy for S7
  bool looked_up = false;                                      // (two driver calls: not on the replay path, where the CPU-side
  auto direct = [&]() -> int {                                 //  latency of the launch is part of every step)
    if (!looked_up) { out_mapped = mapped(out_host); q_mapped = mapped(q_host); looked_up = true; }
    if (!q_mapped) RBQ_CUDA_OK(ctx, cudaMemcpyAsync(dq, q_host, qb, cudaMemcpyHostToDevice, s));
    RBQ_TRY(decode_step_impl(ctx, q_mapped ? q_mapped : dq, q_mapped ? dq : nullptr, cache, idx, p, out_mapped ? out_mapped : dout,
                             nullptr, nullptr, stream));
    if (!out_mapped) RBQ_CUDA_OK(ctx, cudaMemcpyAsync(out_host, dout, ob, cudaMemcpyDeviceToHost, s));
    return RBQ_OK;
  };
  // One CPU-side launch per step instead of seven: the sequence is captured once per argument set and replayed.
  // Not on the legacy default stream (capture is illegal there), not while stage profiling is on (events between kernels).
  if (ctx->prof_on || ctx->host_graph_state < 0 || s == nullptr || s == cudaStreamLegacy || s == cudaStreamPerThread) return direct();
  decltype(ctx->host_key) key;
  memset(&key, 0, sizeof(key));                               // padding bytes take part in the memcmp below
  key.q = q_host; key.out = out_host; key.k = cache->k; key.v = cache->v; key.codes = idx->codes; key.f_scale = idx->f_scale;
  key.f_bias = idx->f_bias; key.c_k = idx->c_k; key.c_q = idx->c_q; key.n_indexed = idx->n_indexed; key.n_total = idx->n_total;
  key.stream = stream; key.ws = ctx->ws; key.sb = (long long)cache->stride_b; key.sh = (long long)cache->stride_h;
  key.st = (long long)cache->stride_t; key.p = p;
  if (ctx->host_graph_state == 1 && memcmp(&key, &ctx->host_key, sizeof(key)) == 0) {
    RBQ_CUDA_OK(ctx, cudaGraphLaunch(ctx->host_graph, s));
    ctx->launches += ctx->host_graph_launches;
    return RBQ_OK;
  }
  if (ctx->host_graph_state == 1) { cudaGraphExecDestroy(ctx->host_graph); ctx->host_graph_state = 0; }
  RBQ_TRY(direct());                                          // this call runs directly (also sets every function attribute)
  const long long l0 = ctx->launches;
  cudaGraph_t g = nullptr;
  if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); ctx->host_graph_state = -1; return RBQ_OK; }
  const int rc = direct();
  const cudaError_t e = cudaStreamEndCapture(s, &g);
  const int nl = (int)(ctx->launches - l0);
  ctx->launches = l0;                                         // captured, not launched
  if (rc != RBQ_OK || e != cudaSuccess || !g || cudaGraphInstantiate(&ctx->host_graph, g, 0) != cudaSuccess) {
    cudaGetLastError();
    if (g) cudaGraphDestroy(g);
    ctx->host_graph_state = -1;
    ctx->err[0] = 0;
    return RBQ_OK;                                            // the direct launch above already did this step
  }
  cudaGraphDestroy(g);
  ctx->host_key = key;
  ctx->host_graph_launches = nl;
  ctx->host_graph_state = 1;
  return RBQ_OK;
}

}  // extern "C"
