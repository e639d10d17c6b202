// rbq_query.cu -- S3 as a stand-alone launch: query pre-processing and INT4 quantisation with its public outputs
// (Alg.2 lines 4-6, L168-172; Eq.5; L524; readings R5/R6/R12 of DESIGN.md).  The arithmetic lives in
// rbq_qprep.cuh; the fused decode step runs the same function inside the estimator CTAs (rbq_estimate.cu), this kernel
// serves rbq_query_quantize / rbq_int4_dot_binary: one CTA per (sequence, KV head), besides the optional public outputs
// (qu, qparams) it writes the private RbqQConst block (B-operand fragments of the estimator MMA, Eq.20 / Eq.2 constants).
#include "rbq_common.cuh"
RBQ_PROBE_DECL(query_probe);
#ifdef RBQ_PROBE
#define RBQ_QPREP_STAMP(slot) do { if (threadIdx.x == 0) RBQ_STAMP(query_probe, slot); } while (0)
#endif
#include "rbq_qprep.cuh"

namespace {

// One CTA per QUERY HEAD, D threads (one rotated coordinate each): S3 is a chain of dependent latencies, and with the G heads
// of a KV group in one CTA the rotation was bound by shared-memory wavefronts (P and the broadcasts of u for two heads per
// thread: 6.3 K cycles of the kernel's 12 K behind its wait; in-kernel stamps, profiles/r02_ncu.md).  A head per CTA reads
// P once and broadcasts one u_i per step; the CTAs of a group share one RbqQConst block and each writes its own part.

template <typename TQ, int D>
__global__ void __launch_bounds__(D)
query_kernel(const TQ* __restrict__ q, const float* __restrict__ c_q, const float* __restrict__ c_k,
             const float* __restrict__ rot, int rot_kind, int Hq, int Hkv, float sm_scale,
             uint8_t* __restrict__ qu_out, float* __restrict__ qparams, RbqQConst* __restrict__ qc_out,
             TQ* __restrict__ q_copy) {
  rbq_pdl_trigger();                               // a dependent S4/S5 launch may become resident while this kernel runs
  if (threadIdx.x == 0) RBQ_STAMP(query_probe, 0);
  extern __shared__ __align__(16) float s_rot[];  // dense, D <= 128: P [D][D], one bulk copy (TMA)
  __shared__ RbqQPrepSmem<D> sm;
  __shared__ __align__(8) unsigned long long s_bar;
  constexpr bool P_SMEM = D <= 128;                 // D = 256: P (256 KB) does not fit, the rotation reads it from L2
  uint32_t bar = 0u;
  if (P_SMEM && rot_kind == RBQ_ROT_DENSE) {
    bar = rbq_smem_u32(&s_bar);
    if (threadIdx.x == 0) {
      rbq_mbar_init(bar, 1);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      rbq_mbar_expect_tx(bar, (uint32_t)(D * D * 4));
      rbq_bulk_g2s(rbq_smem_u32(s_rot), rot, (uint32_t)(D * D * 4), bar);
    }
    __syncthreads();                               // barrier initialised for everyone
  }
  // Launched with programmatic stream serialisation inside the decode step: the launch latency and the copy of P (a
  // constant of the context) overlap the tail of whatever precedes the step on the stream -- in a decode loop the merge
  // phase of the previous step's gather attention, which triggers its dependents when its streaming loop is done.
  // Everything else (q is the caller's, qconst is still read by that step's estimator until its chain has completed)
  // waits here.  Returns at once after an ordinary launch.
  rbq_pdl_wait();
  if (threadIdx.x == 0) RBQ_STAMP(query_probe, 1);
  // blockIdx.x = (sequence b, query head hq) = row of q; its group: (b, hq / G); G is 1, 2 or 4
  const int gsh = (Hq >= 4 * Hkv) ? 2 : (Hq >= 2 * Hkv) ? 1 : 0;
  const int bg = (int)blockIdx.x >> gsh, h0 = (int)blockIdx.x & ((1 << gsh) - 1);
  const int bgs[1] = {bg};
  const int rows0[1] = {(int)blockIdx.x};
  rbq_qprep<TQ, D, 1, P_SMEM>(q, c_q, c_k, rot, s_rot, bar, rot_kind, 1, 1, bgs, rows0, sm_scale, &sm, (int)threadIdx.x, D, 0,
                              qc_out + bg, qu_out, qparams, q_copy, h0, 1 << gsh);
  if (threadIdx.x == 0) RBQ_STAMP(query_probe, 2);
}

template <typename TQ, int D>
int launch_d(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu, float* qparams, void* q_copy, bool pdl, cudaStream_t s) {
  const int BG = ctx->cfg.batch * ctx->cfg.n_q_heads;           // one CTA per query head
  RbqQConst* qc = reinterpret_cast<RbqQConst*>(static_cast<char*>(ctx->ws) + ctx->off_qconst);
  const size_t smem = (ctx->cfg.rot_kind == RBQ_ROT_DENSE && D <= 128) ? (size_t)D * D * sizeof(float) : 0;
  auto kern = query_kernel<TQ, D>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_QUERY + (D == 64 ? 0 : D == 128 ? 1 : 2) * 2 + (sizeof(TQ) == 2 ? 0 : 1), kern, (D <= 128 ? D * D * sizeof(float) : 0));
  if (pdl)
    RBQ_CUDA_OK(ctx, rbq_launch_pdl(kern, dim3(BG), dim3(D), smem, s, (const TQ*)q, (const float*)idx->c_q, (const float*)idx->c_k,
                                    (const float*)ctx->cfg.rot, ctx->cfg.rot_kind, ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads, ctx->sm_scale,
                                    qu, qparams, qc, (TQ*)q_copy));
  else
    kern<<<BG, D, smem, s>>>((const TQ*)q, idx->c_q, idx->c_k, ctx->cfg.rot, ctx->cfg.rot_kind, ctx->cfg.n_q_heads,
                                      ctx->cfg.n_kv_heads, ctx->sm_scale, qu, qparams, qc, (TQ*)q_copy);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

template <typename TQ>
int launch_q(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu, float* qparams, void* q_copy, bool pdl, cudaStream_t s) {
  switch (ctx->cfg.head_dim) {
    case 64: return launch_d<TQ, 64>(ctx, q, idx, qu, qparams, q_copy, pdl, s);
    case 256: return launch_d<TQ, 256>(ctx, q, idx, qu, qparams, q_copy, pdl, s);
    default: return launch_d<TQ, 128>(ctx, q, idx, qu, qparams, q_copy, pdl, s);
  }
}

}  // namespace

int rbq_launch_query(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu, float* qparams, void* q_copy, bool pdl, cudaStream_t s) {
  if (ctx->cfg.q_dtype == RBQ_BF16) return launch_q<__nv_bfloat16>(ctx, q, idx, qu, qparams, q_copy, pdl, s);
  return launch_q<float>(ctx, q, idx, qu, qparams, q_copy, pdl, s);
}

int rbq_probe_copy_query(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, query_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}
