/*
 * rbq.h -- C ABI of the B200-native RaBitQCache decode hot path (arxiv/paper_2606_31519).
 *
 * One library, librbq_b200.so, of hand-written sm_100a CUDA kernels.  Citations are lines of
 * /root/reference/PAPER.md ("L<n>") plus the section / equation / algorithm they fall in.
 *
 * Conventions (all entry points)
 *   - Every call returns int: RBQ_OK (0) or a negative rbq_status.  No exceptions, no exit().
 *     rbq_last_error(ctx) returns a ctx-owned, NUL-terminated description of the last failure.
 *   - ALL tensor arguments are caller-owned DEVICE pointers (allocated by the caller, e.g. with
 *     PyTorch) unless the parameter name ends in `_host`.  The library allocates no device memory
 *     per call; scratch comes from the caller-provided workspace (rbq_workspace_bytes /
 *     rbq_set_workspace).  rbq_config and the rbq_kv / rbq_index structs themselves are HOST
 *     structs holding device pointers; they are read during the call only.
 *   - Calls only ENQUEUE work on the given stream (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and never synchronise the device.  Token counts are read from device
 *     memory (rbq_index.n_indexed / n_total), so no host read-back happens inside a decode step.
 *   - Layouts are row-major and contiguous except K/V, which carry element strides.  head_dim is 64,
 *     128 or 256 (other multiples of 32: RBQ_ERR_UNSUPPORTED).  n_q_heads must be a multiple of n_kv_heads, with
 *     group size G = n_q_heads/n_kv_heads in {1, 2, 4} (8: RBQ_ERR_UNSUPPORTED).  Inputs are assumed finite.
 *   - There is no CPU fallback and no backend dispatch: without a CUDA device every compute call
 *     fails with RBQ_ERR_CUDA.
 *
 * Notation: B sequences, Hq query heads, Hkv KV heads, D = head_dim, Lcap = max_tokens,
 * n_indexed[b] = tokens of sequence b that have codes, n_total[b] = n_indexed[b] + pending.
 */
#ifndef RBQ_H_
#define RBQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rbq_ctx rbq_ctx;

typedef enum {
  RBQ_OK = 0,
  RBQ_ERR_INVALID_ARG = -1,
  RBQ_ERR_UNSUPPORTED = -2,
  RBQ_ERR_WORKSPACE = -3,   /* workspace missing or too small */
  RBQ_ERR_CUDA = -4
} rbq_status;

typedef enum { RBQ_F32 = 0, RBQ_BF16 = 1, RBQ_F16 = 2 /* factor_dtype only */ } rbq_dtype;
typedef enum { RBQ_ROT_DENSE = 0, RBQ_ROT_WH = 1 } rbq_rot_kind;
/* EXACT: canonical fp32 order (R1) -> codes/factors bit-identical to the oracle.
 * FAST : rotation on the tcgen05 tensor cores (bf16 hi/lo split, fp32 accumulate in TMEM: the kernel
 *        takes all 512 TMEM columns of its SM while it runs); codes may differ only where
 *        |y_j| <= 1e-5 ||x||, factors within 1e-5 relative.  Built for bf16 K/V and head_dim 128 (both
 *        rotation kinds: the Walsh-Hadamard rotation runs as its dense matrix); fp32 K/V or head_dim
 *        64 / 256: rbq_create returns RBQ_ERR_UNSUPPORTED. */
typedef enum { RBQ_ENC_EXACT = 0, RBQ_ENC_FAST = 1 } rbq_enc_mode;

/* flags of rbq_encode_keys */
#define RBQ_CK_GIVEN 1u     /* idx->c_k already holds the centroids: do not recompute (L66) */

typedef struct {
  int32_t batch, n_q_heads, n_kv_heads, head_dim;
  int32_t max_tokens;        /* Lcap: capacity per sequence (multiple of 4)                      */
  int32_t flush_tokens;      /* W: pending-window capacity (L215); 0 = never flush              */
  int32_t kv_dtype;          /* rbq_dtype of K/V cache rows                                      */
  int32_t q_dtype;           /* rbq_dtype of q                                                   */
  int32_t out_dtype;         /* rbq_dtype of the attention output                                */
  float sm_scale;            /* softmax scale; 0 => 1/sqrt(head_dim)  (Alg.2 line 12, L184)      */
  int32_t rot_kind;          /* rbq_rot_kind                                                     */
  const float* rot;          /* DEVICE. DENSE: P[D][D] row-major, y_j = sum_i x_i P[i][j] (L149); */
                             /*         WH   : s[D] in {-1,+1}, y = H(s.*x)/sqrt(D), H Sylvester  */
  int32_t enc_mode;          /* rbq_enc_mode                                                     */
  int32_t factor_dtype;      /* rbq_dtype of rbq_index.f_scale: RBQ_F32 (default) or RBQ_F16 -- the paper's 2-byte     */
                             /* correction factor (L752, L756-766: 3.5 % index overhead); the factor is computed in  */
                             /* fp32 exactly as before and rounded to binary16 (RNE) when stored                      */
} rbq_config;

typedef struct {             /* K/V cache; strides in ELEMENTS; one row = D contiguous elements  */
  void* k;                   /* [B][Hkv][Lcap][D] by default                                      */
  void* v;
  int64_t stride_b, stride_h, stride_t;   /* stride_t must be >= D and a multiple of 8           */
} rbq_kv;

typedef struct {
  uint32_t* codes;           /* [B][Hkv][Lcap][D/32]; bit (j%32) of word j/32 = [y_j > 0] (L270, L485) */
  void*     f_scale;         /* [B][Hkv][Lcap] = ||k-c_k||^2 / ||(k-c_k)P||_1 = ||k-c_k|| / <c',P^T k_c> */
                             /*   (Eq.18); 0 when k == c_k; float, or IEEE binary16 when   */
                             /*   factor_dtype = RBQ_F16                                              */
  float*    f_bias;          /* [B][Hq][Lcap] = <c_q[b,h], k_t> (L89); NULL iff c_q is NULL      */
  float*    c_k;             /* [B][Hkv][D] key centroids (Alg.1 line 4, L116)                   */
  const float* c_q;          /* [B][Hq][D] query centroids or NULL (= zero centroid)             */
  int32_t*  n_indexed;       /* [B]                                                              */
  int32_t*  n_total;         /* [B]                                                              */
} rbq_index;

/* ---- context ------------------------------------------------------------------------------ */
/* Validates the config and creates a context (host object; owns two CUDA events and a small
 * device block of per-query constants carved from the workspace).                              */
int rbq_create(const rbq_config* cfg_host, rbq_ctx** out);
int rbq_destroy(rbq_ctx* ctx);
/* Bytes of device scratch the calls below need for this config (query constants, Top-p state,
 * split-K attention partials, scores of the fused step).                                       */
int rbq_workspace_bytes(const rbq_ctx* ctx, size_t* bytes);
/* `dev` must stay valid and 256-byte aligned until rbq_destroy or the next rbq_set_workspace.  Setup call: clears the
 * 4-byte device status word with a blocking cudaMemset and drops the CUDA graph of rbq_decode_step_host, if any.      */
int rbq_set_workspace(rbq_ctx* ctx, void* dev, size_t bytes);
/* Sticky device-side status bits.  RBQ_FLAG_APPEND_OVERFLOW: an rbq_append_tokens call asked for rows beyond max_tokens;
 * those rows were dropped and n_total clamped to max_tokens (nothing was written out of bounds).  BLOCKS: copies the
 * word to flags_host on `stream` and synchronises that stream (like rbq_profile_read, not part of a decode step).     */
#define RBQ_FLAG_APPEND_OVERFLOW 1u
int rbq_status_flags(rbq_ctx* ctx, uint32_t* flags_host, void* stream);
const char* rbq_last_error(const rbq_ctx* ctx);

/* ---- S1  Alg.1 index construction (L106-147, L149-151, L485-487) ---------------------------- */
/* For every (b, kv head) encodes tokens [0, seq_lens[b]): c_k = mean of those keys (unless
 * RBQ_CK_GIVEN), x = k - c_k, y = x P, codes = packed [y > 0], f_scale = ||x||^2/||y||_1,
 * f_bias = <c_q, k> when c_q != NULL.  Sets n_indexed = n_total = seq_lens.  seq_lens: DEVICE [B]. */
int rbq_encode_keys(rbq_ctx* ctx, const rbq_kv* cache, const int32_t* seq_lens, uint32_t flags,
                    rbq_index* idx, void* stream);

/* ---- S2/S8  lazy decode updates (L215; R14) --------------------------------------- */
/* k_new, v_new: [B][Hkv][n_new][D] contiguous, kv_dtype.  (1) if an earlier call enqueued a flush,
 * `stream` waits for it and n_indexed += flushed; (2) rows are copied to cache rows
 * [n_total, n_total+n_new), n_total += n_new; (3) if pending >= W, the oldest floor(pending/W)*W
 * pending rows are encoded with the frozen c_k on `side_stream` (ordered after the copy by an
 * event); they stay pending until the next rbq_append_tokens call.  side_stream may equal stream.
 * Every sequence of the batch appends the same n_new rows per call (the pending count is uniform over the batch and
 * is shadowed on the host); rows that would exceed max_tokens are dropped and flagged (rbq_status_flags).            */
int rbq_append_tokens(rbq_ctx* ctx, const void* k_new, const void* v_new, int32_t n_new,
                      rbq_kv* cache, rbq_index* idx, void* stream, void* side_stream);

/* ---- S3  query pre-processing + INT4 quantisation (Alg.2 lines 4-6, L168-172; Eq.5; L524) */
/* q: [B][Hq][D] q_dtype.  Optional outputs (each may be NULL): qu uint8 [B][Hq][D] in [0,15];
 * qparams float [B][Hq][6] = {||q-c_q||, q_l, Delta, sum(qu), <q,c_k>, <c_q,c_k>}.
 * Always refreshes the context's private query constants used by S4/S5.                        */
int rbq_query_quantize(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu,
                       float* qparams, void* stream);

/* ---- S4  Int4_Dot_Binary (Alg.2 line 8, L176; L268-274; L534) -------------------------------- */
/* dot[b][h][t] = <c_b[t], qu[b][h]> (exact integer), pop[b][g][t] = popcount(c_b[t]) for
 * t < n_indexed[b]; int32 [B][Hq][Lcap] / [B][Hkv][Lcap].  Includes S3.                         */
int rbq_int4_dot_binary(rbq_ctx* ctx, const void* q, const rbq_index* idx, int32_t* dot,
                        int32_t* pop, void* stream);

/* ---- S3-S5  estimated logits (Alg.2 lines 4-10; Eq.20, Eq.18, Eq.2) ------------ */
/* scores[b][h][t] = sm_scale * ( ||q-c_q|| f_scale[t] (2 Delta dot + 2 q_l pop - Delta sum(qu)
 * - D q_l) + <q,c_k> + f_bias[t] - <c_q,c_k> ) for t < n_indexed[b]; float [B][Hq][Lcap].       */
int rbq_estimate_scores(rbq_ctx* ctx, const void* q, const rbq_index* idx, float* scores,
                        void* stream);

/* ---- S6  adaptive Top-p selection (Alg.2 line 12, L184, L201) -------------------------------- */
/* Per row (b,h): the minimal set I whose softmax mass over t < n_indexed[b] is >= p, ties broken
 * towards the lowest index; p >= 1 selects every indexed token.  sel_idx int32 [B][Hq][Lcap]
 * (first sel_cnt[b][h] entries valid, ascending token order), sel_cnt int32 [B][Hq].            */
int rbq_topp_select(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p,
                    int32_t* sel_idx, int32_t* sel_cnt, void* stream);

/* The same operation (same kernels, same results bit for bit) for callers that cannot allocate device memory or hand over
 * a workspace (code under CUDA graph capture, tight serving loops): needs NO workspace (rbq_set_workspace may never have been
 * called) and calls no cudaMalloc / cudaFree / allocating routine.  Its scratch -- the row-maximum keys and the per-row
 * selection bitmaps, 4 * (roundup(B*Hq, 64) + B*Hq * roundup(ceil(Lcap/32), 4)) bytes -- lives in ONE static device array
 * of 2 MiB inside the library (every GPU that loads the library holds it until exit), so
 *   B*Hq * (Lcap/32 + 1)  must stay below 524 288 words (e.g. 32 rows x 131 072 tokens; 128 rows x 65 536 tokens);
 * beyond that: RBQ_ERR_UNSUPPORTED with the sizes in rbq_last_error -- use rbq_topp_select.  All calls (all contexts of the
 * process on one device) share the array: it keeps the last call's contents (what must start at zero is cleared per call),
 * and two calls that overlap on the GPU (different streams, no ordering) race.  Arguments, layouts, ownership and the
 * other errors as for rbq_topp_select; asynchronous on `stream`.                                                      */
int rbq_topp_select_static(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p,
                           int32_t* sel_idx, int32_t* sel_cnt, void* stream);

/* ---- S6'  the paper's Top-p operator: Algorithm 3, ternary threshold search (L217-252; 4.1 L256-264;
 *           App. B.1) -- alternative selector, SURVEY.md 8(f) row 2 --------------------- */
/* Per row: prob = softmax(scores[b][h][0..n_indexed[b])) in fp64; low = 0, high = max(prob); repeat
 * { pi0 = (high + 2 low)/3, pi1 = (2 high + low)/3, G0/G1 = mass above pi0/pi1, v_min = min{s > low},
 * v_max = max{s <= high}; G1 >= p: low = pi1; else G0 >= p: low = pi0, high = min(pi1, v_max); else
 * high = min(pi0, v_max) } until v_min = v_max (at most 4096 iterations); selected = {t : prob_t > low}.
 * Unlike rbq_topp_select this keeps EVERY token tied with the boundary value (Alg.3's mask), so the set
 * is the minimal one only when the boundary value is unique.  p >= 1 selects every indexed token.
 * Same buffers as rbq_topp_select (device pointers; sel_idx ascending); iters int32 [B][Hq] or NULL
 * receives the iteration counts.  Needs no workspace.  Rows longer than 204 800 tokens:
 * RBQ_ERR_UNSUPPORTED.                                                                            */
int rbq_topp_select_alg3(rbq_ctx* ctx, const float* scores, const rbq_index* idx, float p,
                         int32_t* sel_idx, int32_t* sel_cnt, int32_t* iters, void* stream);

/* ---- S7  hybrid attention over selected U pending tokens (Alg.2 lines 14-15, L188-190, L215) -- */
/* out[b][h] = sum_{t in A} softmax_A(<q,k_t> sm_scale)_t v_t, A = sel_idx[b][h][0..cnt) U
 * [n_indexed[b], n_total[b]); out_dtype [B][Hq][D]; lse float [B][Hq] or NULL (log-sum-exp over A).
 * Empty A gives out = 0, lse = -inf.
 * Summation order (the paper fixes none, R19): with bf16 K/V and q and head_dim <= 128 the rows of a KV group are
 * handed to the warps of the GPU dynamically, so the fp32 accumulation order -- not the attended set -- varies from call to
 * call and two calls agree to rounding (~1e-6 of the output scale), not bit for bit.  RBQ_GATHER_PLAN=1 in the environment
 * when the context is created selects a static partition (bit-reproducible, one more kernel launch); fp32 inputs and
 * head_dim 256 always take a static partition.  Calls on one context must not overlap on the GPU (shared workspace:
 * selection bitmaps, per-group counters).                                                        */
int rbq_sparse_attention(rbq_ctx* ctx, const void* q, const rbq_kv* cache, const rbq_index* idx,
                         const int32_t* sel_idx, const int32_t* sel_cnt, void* out, float* lse,
                         void* stream);

/* ---- fused decode step: S3 -> S4/S5 -> S6 -> S7 (Alg.2) ---------------------------- */
/* sel_idx / sel_cnt are optional outputs.  Internally the selection is a per-row bitmap in the
 * workspace; sel_idx == NULL skips materialising the index lists (2.4 MB of writes at config 2). */
int rbq_decode_step(rbq_ctx* ctx, const void* q, const rbq_kv* cache, const rbq_index* idx, float p,
                    void* out, int32_t* sel_idx, int32_t* sel_cnt, void* stream);

/* ---- host-buffer convenience used by the end-to-end measurement ------------------------------ */
/* Same as rbq_decode_step but q_host / out_host are HOST buffers (pinned recommended): copies q
 * host->device, runs the step, copies out device->host, all on `stream`; staging device buffers
 * come from the workspace.  With page-locked (mapped) buffers the copies disappear: S3 reads
 * q_host over PCIe (leaving a device copy for S7) and the last kernel stores the result straight
 * into out_host; pageable buffers are staged with cudaMemcpyAsync.  Does not synchronise; the
 * caller synchronises the stream (the result is valid in out_host only after that).  On a
 * non-default stream the sequence is captured once per argument set and replayed as one CUDA graph
 * (one CPU-side launch per step); on the legacy default stream it is launched directly.        */
int rbq_decode_step_host(rbq_ctx* ctx, const void* q_host, const rbq_kv* cache, const rbq_index* idx,
                         float p, void* out_host, void* stream);

/* Number of kernel launches the library has enqueued through this context so far.              */
int64_t rbq_launch_count(const rbq_ctx* ctx);

/* ---- per-stage device timing of rbq_decode_step (measurement aid) ----------------- */
/* Stages: 0 = S3 query prep, 1 = S4/S5 estimator, 2 = S6 Top-p, 3 = S7 union plan (a launch of its own only on the
 * static-partition paths: 0 ms when the gather expands the selection bitmaps itself), 4 = S7 gather attention (including
 * the merge of its partials).  While enabled, every rbq_decode_step records RBQ_N_STAGES + 1 timing
 * events on its stream (up to RBQ_PROFILE_MAX_STEPS steps, later steps are not recorded).
 * rbq_profile_read BLOCKS until the recorded steps have finished (the only call that waits),
 * writes the summed milliseconds per stage to ms_host[RBQ_N_STAGES] and the number of recorded
 * steps to n_steps_host, and clears the record.                                                  */
#define RBQ_N_STAGES 5
#define RBQ_PROFILE_MAX_STEPS 512
int rbq_profile_enable(rbq_ctx* ctx, int enable);
int rbq_profile_read(rbq_ctx* ctx, float* ms_host, int32_t* n_steps_host);

/* ---- in-kernel timeline probes (measurement aid; only in the probe build of the library) ------------------------------ */
/* `python -m paper_2606_31519_b200.build --probe` builds librbq_b200_probe.so with -DRBQ_PROBE: its kernels stamp clock64
 * of chosen points (slot 15: %globaltimer of slot 0) into a device buffer [256 CTAs][16 slots] per kernel.  kernel: 0 =
 * estimator, 1 = Top-p, 2 = gather attention, 3 = union plan, 4 = query preparation.  BLOCKS (device synchronise + copy) and writes 256 * 16
 * uint64 to out_host.  The regular library returns RBQ_ERR_UNSUPPORTED.                                             */
int rbq_probe_dump(rbq_ctx* ctx, int kernel, uint64_t* out_host);

/* ---- row-gather experiment (measurement aid, hard part 5; Alg.2 line 14: the gather of the
 * selected K / V rows) --------------------------------------------------------------------------------------------------- */
/* Streams the rows rows[0 .. n) (device, int32, each in [0, n_rows_total)) of two bf16 matrices K and V (device,
 * [n_rows_total][128], contiguous 256-byte rows) through shared memory with the launch shape and pipeline depth of the gather
 * attention kernel (one persistent CTA per SM, 8 warps x 3 stages x 16-row K + V tiles) and adds the sum of all gathered
 * 32-bit words to *checksum (device, uint64, NOT cleared by the call).  mode 0: 16-byte cp.async per lane (what S7 uses);
 * mode 1: TMA cp.async.bulk.tensor.2d tile::gather4, four rows per instruction; modes 2 / 3: the same two with K pointing at
 * ONE matrix of interleaved K | V rows ([n_rows_total][256], 512-byte rows; V is ignored and may be NULL).  Asynchronous on
 * `stream`; nothing of the context's state is touched.  Errors: RBQ_ERR_INVALID_ARG, RBQ_ERR_UNSUPPORTED (no tensor-map
 * entry point in the driver), RBQ_ERR_CUDA.                                                                            */
int rbq_diag_gather(rbq_ctx* ctx, const void* K, const void* V, long long n_rows_total, const int32_t* rows, long long n,
                    int mode, unsigned long long* checksum, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* RBQ_H_ */
