// rbq_common.cuh -- shared host/device declarations of the B200 RaBitQCache library.
// CUDA path only: nothing here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/rbq.h"

#define RBQ_D 128            // head_dim of the kernels that are not templated on it yet
#define RBQ_WORDS 4          // D/32 code words per token at D = 128
#define RBQ_MAX_G 4          // query heads per KV head (N=8 MMA columns: G heads + G ones-columns)
#define RBQ_MAX_KSTEPS 8     // k-steps of the estimator MMA: D/32 (2, 4, 8 for D = 64, 128, 256)

// Private per-(sequence, KV head) query constants produced by S3 and consumed by S4/S5.
// bfrag: B-operand fragments of mma.m16n8k32.u8 in register order [k-step][lane][2]
//        (column 2j = query head j of the group, column 2j+1 = all-ones -> popcount),
//        pre-scaled by 2^(3-n) so that the masked code bytes (value 2^n) need no shift.
//        Which code bit a (k-step, lane, register, byte) position stands for: rbq_bfrag_dim below.
struct __align__(16) RbqQConst {
  uint32_t bfrag[RBQ_MAX_KSTEPS][32][2];
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
      off_stage_q, off_stage_out, off_centroid, off_gnext, off_rho, off_uexact, total_bytes;
  int gather_via_plan;       // RBQ_GATHER_PLAN=1 in the environment at rbq_create: S7 through attn_plan_kernel + union lists (deterministic
                             // accumulation order) instead of straight from the bitmaps
  cudaEvent_t ev_copy, ev_flush;
  unsigned char attr_done[128];   // kernel instantiations whose MaxDynamicSharedMemorySize was set for THIS context's device (RBQ_ATTR_*)
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

// per-context "function attribute set" slots (the attribute is per device; a context lives on one device): base ids, each
// kernel family adds the index of its instantiation
enum { RBQ_ATTR_QUERY = 0 /* +6 */, RBQ_ATTR_EST = 8 /* +36 */, RBQ_ATTR_TOPP = 48 /* +9 */, RBQ_ATTR_ENC_EXACT = 60 /* +12 */,
       RBQ_ATTR_FBIAS = 74 /* +6 */, RBQ_ATTR_ENC_FAST = 82, RBQ_ATTR_GATHER = 84 /* +8 */, RBQ_ATTR_ALG3 = 94, RBQ_ATTR_MISC = 96 };

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
// the per-token factor as stored: fp32, or binary16 (RNE) when rbq_config.factor_dtype = RBQ_F16
__device__ __forceinline__ void rbq_store_factor(void* f_scale, int f16, size_t i, float v) {
  if (f16) reinterpret_cast<__half*>(f_scale)[i] = __float2half_rn(v);
  else reinterpret_cast<float*>(f_scale)[i] = v;
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

// ---- estimator operand layout (shared by S3, which builds the B fragments, and S4, which builds the A fragments) ------
// A fragment of mma.m16n8k32.u8 held by lane (g, tp): register r of k-step s holds 4 bytes, byte i <-> k = 4 tp + i (+16 for
// r = 1).  The 1-bit code of a token is expanded to those bytes by masking a 32-bit value x that lane tp derives from the
// token's code words (W = D/32 words per token):
//   W = 4: x = word tp;                       byte i of register (s, r): bit e = 2 s + r of code byte i of x      (value 2^(e & 3))
//   W = 8: x_u = word 2 tp + u, u = s >> 2;   same with s' = s & 3
//   W = 2: v = 16-bit half (tp & 1) of word tp >> 1, x = v | (v >> 1) << 16; bit e' = 4 s + 2 r of x's byte i  (value 2^(2 r)),
//          i.e. code bit e' + (i >> 1) of code byte 2 (tp & 1) + (i & 1)
// Returns the head dimension that position multiplies and the left shift that makes (A byte) * (B byte) = 8 * bit * qu.
__host__ __device__ inline void rbq_bfrag_dim(int W, int s, int tp, int r, int i, int& dim, int& shift) {
  if (W == 2) {
    const int e = 4 * s + 2 * r;
    dim = 32 * (tp >> 1) + 8 * (2 * (tp & 1) + (i & 1)) + e + (i >> 1);
    shift = 3 - 2 * r;
  } else {
    const int u = (W == 8) ? (s >> 2) : 0, sp = s & 3, e = 2 * sp + r;
    dim = 32 * ((W == 8 ? 2 * tp : tp) + u) + 8 * i + e;
    shift = 3 - (e & 3);
  }
}

// ---- mbarrier / bulk-copy (TMA, UBLKCP) helpers ------------------------------------------------------------------------
__device__ __forceinline__ uint32_t rbq_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void rbq_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void rbq_mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void rbq_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void rbq_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// bounded spin on a phase parity: a protocol mistake must trap, not hang the GPU
__device__ __forceinline__ void rbq_mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  for (uint32_t spin = 0; !done; ++spin) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (spin > (1u << 22)) __trap();
  }
}
// 1-D bulk copy global -> shared (bytes a multiple of 16, both addresses 16-byte aligned), completion on an mbarrier
__device__ __forceinline__ void rbq_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar) : "memory");
}

// ---- in-kernel timeline probes (build option: python -m paper_2606_31519_b200.build --probe -> librbq_b200_probe.so) -----
// With -DRBQ_PROBE a kernel stamps clock64 (and %globaltimer in the slot after it) of chosen points into a per-file device
// buffer [RBQ_PROBE_CTAS][RBQ_PROBE_SLOTS]; rbq_probe_dump(kernel id) copies it out.  Without the flag the macros vanish.
#define RBQ_PROBE_CTAS 256
#define RBQ_PROBE_SLOTS 16
enum { RBQ_PROBE_ESTIMATE = 0, RBQ_PROBE_TOPP = 1, RBQ_PROBE_GATHER = 2, RBQ_PROBE_PLAN = 3, RBQ_PROBE_QUERY = 4, RBQ_PROBE_KERNELS = 5 };
#ifdef RBQ_PROBE
#define RBQ_PROBE_DECL(name) __device__ unsigned long long name[RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS]
#define RBQ_STAMP(buf, slot)                                                                                   \
  do {                                                                                                         \
    if (blockIdx.x < RBQ_PROBE_CTAS) {                                                                         \
      (buf)[blockIdx.x * RBQ_PROBE_SLOTS + (slot)] = (unsigned long long)clock64();                            \
      if ((slot) == 0) {                          /* the global timer only once: reading it is slow */           \
        unsigned long long gt_;                                                                                \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_));                                                \
        (buf)[blockIdx.x * RBQ_PROBE_SLOTS + RBQ_PROBE_SLOTS - 1] = gt_;                                       \
      }                                                                                                        \
    }                                                                                                          \
  } while (0)
#else
#define RBQ_PROBE_DECL(name)
#define RBQ_STAMP(buf, slot) do {} while (0)
#endif
int rbq_probe_copy_estimate(unsigned long long* host);      // defined in the .cu that owns the buffer; RBQ_ERR_UNSUPPORTED without RBQ_PROBE
int rbq_probe_copy_topp(unsigned long long* host);
int rbq_probe_copy_gather(unsigned long long* host);
int rbq_probe_copy_plan(unsigned long long* host);
int rbq_probe_copy_query(unsigned long long* host);

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
#define RBQ_SET_SMEM_ATTR(ctx, id, func, bytes)                                                           \
  do {                                                                                                    \
    if (!(ctx)->attr_done[(id)]) {                                                                        \
      RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes))); \
      (ctx)->attr_done[(id)] = 1;                                                                         \
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
// pdl: launched with programmatic stream serialisation (the kernel waits for its predecessor before it reads q or writes)
int rbq_launch_query(rbq_ctx*, const void* q, const rbq_index*, uint8_t* qu, float* qparams, void* q_copy, bool pdl, cudaStream_t);
// S4/S5 behind an rbq_launch_query.  rowmax_key: zeroed keys that receive the row maxima, or NULL.
int rbq_launch_estimate(rbq_ctx*, const rbq_index*, float* scores, int32_t* dot, int32_t* pop, uint32_t* rowmax_key, cudaStream_t);
// S6 writes the per-row selection bitmap sel_bits [B*Hq][rbq_words_per_row] (always), sel_cnt, and sel_idx if non-NULL.
// rowmax_key: order-preserving keys of the row maxima [B*Hq] (written by S5), or NULL to compute them here.
int rbq_topp_init(rbq_ctx* ctx);   // uploads the Top-p kernel's fp64 tables (once per context)
// S6 on caller-provided scores with its scratch in a static device array (no workspace, no allocation; rbq_topp.cu)
int rbq_launch_topp_static(rbq_ctx*, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx, int32_t* sel_cnt,
                           cudaStream_t);
int rbq_launch_topp(rbq_ctx*, const float* scores, uint32_t* rowmax_key, const int32_t* n_indexed, float p,
                    uint32_t* sel_bits, int32_t* sel_idx, int32_t* sel_cnt, cudaStream_t);
// Alg.3 selector (ternary threshold search in fp64): ascending sel_idx, sel_cnt, optional iteration counts [B*Hq].
int rbq_launch_topp_alg3(rbq_ctx*, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx, int32_t* sel_cnt,
                         int32_t* iters, cudaStream_t);
int rbq_launch_bits_from_lists(rbq_ctx*, const rbq_index*, const int32_t* sel_idx, const int32_t* sel_cnt,
                               uint32_t* sel_bits, cudaStream_t);
// S7 from the selection bitmaps: union plan -> gather attention -> merge.
// sel_cnt: per-row selection counts (device): the bitmap-driven gather sizes its work partition with them.
int rbq_launch_attention(rbq_ctx*, const void* q, const RbqKV&, const rbq_index*, const uint32_t* sel_bits,
                         const int32_t* sel_cnt, void* out, float* lse, cudaStream_t);
size_t rbq_attention_part_bytes(const rbq_ctx*);
bool rbq_attention_from_bits(const rbq_ctx*);   // bf16 tensor-pipe gather that expands the bitmaps itself (needs the union sizes)
// 32-bit words per bitmap row, padded to a multiple of 4 (16-byte vector loads)
static inline int rbq_words_per_row(const rbq_ctx* c) { return (((c->cfg.max_tokens + 31) / 32) + 3) & ~3; }
