// rbq_common.cuh -- shared host/device declarations of the B200 RaBitQCache library.
// CUDA path only: nothing here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/rbq.h"

#define RBQ_D 128            // head_dim supported by every kernel
#define RBQ_WORDS 4          // D/32 code words per token
#define RBQ_MAX_G 4          // query heads per KV head (N=8 MMA columns: G heads + G ones-columns)

// Private per-(sequence, KV head) query constants produced by S3 and consumed by S4/S5.
// bfrag: B-operand fragments of mma.m16n8k32.u8 in register order [k-step][lane][2]
//        (column 2j = query head j of the group, column 2j+1 = all-ones -> popcount),
//        pre-scaled by 2^(3-n) so that the masked code bytes (value 2^n) need no shift.
struct __align__(16) RbqQConst {
  uint32_t bfrag[4][32][2];
  float cA[RBQ_MAX_G];       // sm_scale * ||q-c_q|| * Delta / 4
  float cB[RBQ_MAX_G];       // sm_scale * ||q-c_q|| * q_l   / 4
  float cD[RBQ_MAX_G];       // sm_scale * (<q,c_k> - <c_q,c_k>)
  int32_t init_d[RBQ_MAX_G]; // 0x4B400000 - 4*sum(qu): accumulator start (float-magic biased)
  int32_t init_p;            // 0x4B400000 - 4*D
  int32_t pad[3];
};

struct RbqKV {               // device view of rbq_kv
  const void* k;
  const void* v;
  long long sb, sh, st;      // element strides
};

struct rbq_ctx {
  rbq_config cfg;
  int G;
  float sm_scale;
  int sm_count;
  void* ws;
  size_t ws_bytes;
  // workspace carve-up (byte offsets), filled by rbq_layout_workspace
  size_t off_qconst, off_scores, off_selbits, off_selcnt, off_ulist, off_ucount, off_gdone, off_rowmax, off_part,
      off_stage_q, off_stage_out, off_centroid, total_bytes;
  cudaEvent_t ev_copy, ev_flush;
  unsigned attr_mask;        // kernels whose MaxDynamicSharedMemorySize was set for THIS context's device (RBQ_ATTR_*)
  size_t attr_topp_smem;     // largest dynamic shared memory size set for the Top-p kernels so far
  size_t off_flags;          // device status word (RBQ_FLAG_*), sticky
  int pending;               // host shadow of n_total - n_indexed (uniform over the batch: every sequence appends n_new rows per call)
  int in_flight;             // rows encoded by an enqueued flush, not yet committed
  long long launches;
  int prof_on, prof_steps;                                   // stage timing (rbq_profile_*)
  cudaEvent_t* stage_ev;                                     // events of the step being enqueued, or NULL
  cudaEvent_t* prof_ev;                                      // [RBQ_PROFILE_MAX_STEPS][RBQ_N_STAGES + 1], lazily created
  // rbq_decode_step_host: the copies and the five launches replayed as one CUDA graph while the arguments stay the same
  cudaGraphExec_t host_graph;
  int host_graph_state;      // 0 = none yet, 1 = valid, -1 = capture not possible on this stream / driver: direct launches
  int host_graph_launches;   // kernel launches one replay stands for
  struct { const void *q, *out, *k, *v, *codes, *f_scale, *f_bias, *c_k, *c_q, *n_indexed, *n_total, *stream, *ws;
           long long sb, sh, st; float p; } host_key;
  char err[256];
};

// per-context "function attribute set" bits (the attribute is per device; a context lives on one device)
enum { RBQ_ATTR_QUERY = 1u, RBQ_ATTR_ENC_EXACT = 2u, RBQ_ATTR_ENC_FAST = 4u, RBQ_ATTR_GATHER = 8u, RBQ_ATTR_ALG3 = 16u,
       RBQ_ATTR_EST = 32u, RBQ_ATTR_FUSED = 64u };

#define RBQ_FAIL(ctx, code, ...)                                   \
  do {                                                             \
    if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__); \
    return (code);                                                 \
  } while (0)

#define RBQ_CUDA_OK(ctx, expr)                                                      \
  do {                                                                              \
    cudaError_t e_ = (expr);                                                        \
    if (e_ != cudaSuccess) RBQ_FAIL(ctx, RBQ_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

#define RBQ_LAUNCH_OK(ctx)                                                          \
  do {                                                                              \
    cudaError_t e_ = cudaGetLastError();                                            \
    if (e_ != cudaSuccess) RBQ_FAIL(ctx, RBQ_ERR_CUDA, "launch failed at %s:%d: %s", __FILE__, __LINE__, cudaGetErrorString(e_)); \
    (ctx)->launches++;                                                              \
  } while (0)

// ---- device helpers ---------------------------------------------------------------------------
__device__ __forceinline__ float rbq_ld_elem(const float* p, long long i) { return p[i]; }
__device__ __forceinline__ float rbq_ld_elem(const __nv_bfloat16* p, long long i) {
  return __bfloat162float(p[i]);
}
__device__ __forceinline__ void rbq_st_elem(float* p, long long i, float v) { p[i] = v; }
__device__ __forceinline__ void rbq_st_elem(__nv_bfloat16* p, long long i, float v) {
  p[i] = __float2bfloat16_rn(v);
}
__device__ __forceinline__ float rbq_bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float rbq_bf16hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// order-preserving map float -> uint32 (larger float <=> larger key)
__device__ __forceinline__ uint32_t rbq_fkey(float f) {
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float rbq_fkey_inv(uint32_t k) {
  uint32_t u = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
  return __uint_as_float(u);
}

// ---- programmatic dependent launch (PDL) -----------------------------------------------------------
// The kernels of a decode step are launched with programmatic stream serialisation: a kernel's CTAs may become
// resident while its predecessor drains, which hides the launch latency between the short kernels of the step.
// Every kernel calls rbq_pdl_trigger() first and rbq_pdl_wait() before it touches anything the predecessor
// wrote (and before any early exit, so that completion stays transitive along the chain).
__device__ __forceinline__ void rbq_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void rbq_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t rbq_launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// MaxDynamicSharedMemorySize is a per-device attribute of a function: it is set once per CONTEXT (a context lives on the
// device that was current at rbq_create), always to the same per-kernel maximum, so that contexts with different
// configurations on one device never lower each other's limit.
#define RBQ_SET_SMEM_ATTR(ctx, bit, func, bytes)                                                          \
  do {                                                                                                    \
    if (!((ctx)->attr_mask & (bit))) {                                                                    \
      RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes))); \
      (ctx)->attr_mask |= (bit);                                                                          \
    }                                                                                                     \
  } while (0)
#define RBQ_MAX_DYN_SMEM (227 * 1024)


// ---- kernel launchers (defined in the .cu files, called from rbq_api.cu) ------------------------
int rbq_launch_centroid(rbq_ctx*, const RbqKV&, const int32_t* seq_lens, float* c_k, cudaStream_t);
int rbq_launch_encode(rbq_ctx*, const RbqKV&, const int32_t* t_begin, const int32_t* t_count_or_null,
                      int fixed_count, int max_count, const rbq_index*, cudaStream_t);
int rbq_launch_encode_fast(rbq_ctx*, const RbqKV&, const int32_t* t_begin, const int32_t* t_count_or_null,
                           int fixed_count, int max_count, const rbq_index*, cudaStream_t);   // RBQ_ENC_FAST, bf16 K, dense P
int rbq_launch_set_counts(rbq_ctx*, const int32_t* seq_lens, int32_t* n_indexed, int32_t* n_total,
                          cudaStream_t);
int rbq_launch_append_copy(rbq_ctx*, const void* k_new, const void* v_new, int n_new, const RbqKV&,
                           int32_t* n_indexed, int32_t* n_total, int commit, cudaStream_t);
// q_copy (or NULL): device buffer that receives a verbatim copy of q (used when q lives in mapped host memory)
int rbq_launch_query(rbq_ctx*, const void* q, const rbq_index*, uint8_t* qu, float* qparams, void* q_copy, cudaStream_t);
int rbq_launch_estimate(rbq_ctx*, const rbq_index*, float* scores, int32_t* dot, int32_t* pop,
                        cudaStream_t);
// S6 writes the per-row selection bitmap sel_bits [B*Hq][rbq_words_per_row] (always), sel_cnt, and sel_idx if non-NULL.
// rowmax_key: order-preserving keys of the row maxima [B*Hq] (written by S5), or NULL to compute them here.
int rbq_launch_topp(rbq_ctx*, const float* scores, const uint32_t* rowmax_key, const int32_t* n_indexed, float p,
                    uint32_t* sel_bits, int32_t* sel_idx, int32_t* sel_cnt, cudaStream_t);
// Alg.3 selector (ternary threshold search in fp64): ascending sel_idx, sel_cnt, optional iteration counts [B*Hq].
int rbq_launch_topp_alg3(rbq_ctx*, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx, int32_t* sel_cnt,
                         int32_t* iters, cudaStream_t);
int rbq_launch_bits_from_lists(rbq_ctx*, const rbq_index*, const int32_t* sel_idx, const int32_t* sel_cnt,
                               uint32_t* sel_bits, cudaStream_t);
// S7 from the selection bitmaps: union plan -> gather attention -> merge.
int rbq_launch_attention(rbq_ctx*, const void* q, const RbqKV&, const rbq_index*, const uint32_t* sel_bits,
                         void* out, float* lse, cudaStream_t);
size_t rbq_attention_part_bytes(const rbq_ctx*);
// 32-bit words per bitmap row, padded to a multiple of 4 (16-byte vector loads)
static inline int rbq_words_per_row(const rbq_ctx* c) { return (((c->cfg.max_tokens + 31) / 32) + 3) & ~3; }
