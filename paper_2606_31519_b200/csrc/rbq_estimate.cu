// rbq_estimate.cu -- S4 + S5: binary x INT4 proxy logits over the whole indexed context
// (Alg.2 lines 8-10, L176-180; L268-274; Eq.20; Eq.18; Eq.2).
//
// Design (B200, sm_100a).  Per (token, KV head) the method must move 16 B of code + 4 B of f_scale;
// the G query heads of the group share that stream.  Plain AND+POPC needs 16*G POPC per token and
// is bound by the 16 lanes/clk/SM POPC pipe (measured), ~5x over the HBM time, so the integer dot
// runs on the tensor pipe instead: the 1-bit code is expanded IN REGISTERS to u8 operands with ONE
// LOP3 per 4 dims (w & (0x01010101 << n) keeps bit n of every byte at value 2^n; the u8 query
// operand is pre-scaled by 2^(3-n), so no shift is needed and the s32 accumulator holds 8*<c_b,qu>),
// and mma.sync.m16n8k32.u8.u8.s32 (native IMMA.16832 on sm_100a) contracts 16 tokens x 128 dims
// against 8 columns = G query heads interleaved with all-ones columns (the latter yield
// 8*popcount(c_b) for free).  The K permutation implied by the masks is baked into the B fragments
// by S3.  Codes and factors are staged HBM -> shared memory by TMA bulk copies (cp.async.bulk +
// mbarrier), all stages of a CTA in flight at once; warps consume 32-token groups.
//
// Integer results are exact.  Epilogue in fp32 without cancellation:
//   acc_d = 4*(2*dot - sum(qu)), acc_p = 4*(2*pop - D)   (exact ints: accumulators start at
//   0x4B400000 - 4*sum(qu) / - 4*D, so reinterpreting as float and subtracting 2^23+2^22 converts)
//   score = f_scale*(cA*acc_d + cB*acc_p) + cD [+ sm_scale*f_bias].
#include "rbq_common.cuh"

namespace {

constexpr int EST_THREADS = 256;
constexpr int EST_STAGES = 4;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LAB_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra LAB_DONE_%=;\n"
      "bra LAB_WAIT_%=;\n"
      "LAB_DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

__device__ __forceinline__ void imma_16832(int (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                           uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// One 16-token tile: rows g (code word wa) and g+8 (code word wb) of this lane's quad column.
__device__ __forceinline__ void tile_mma(int (&c)[4], uint32_t wa, uint32_t wb, const uint32_t (&bf)[4][2]) {
  const uint32_t ha = wa >> 4, hb = wb >> 4;
  imma_16832(c, wa & 0x01010101u, wb & 0x01010101u, wa & 0x02020202u, wb & 0x02020202u, bf[0][0], bf[0][1]);
  imma_16832(c, wa & 0x04040404u, wb & 0x04040404u, wa & 0x08080808u, wb & 0x08080808u, bf[1][0], bf[1][1]);
  imma_16832(c, ha & 0x01010101u, hb & 0x01010101u, ha & 0x02020202u, hb & 0x02020202u, bf[2][0], bf[2][1]);
  imma_16832(c, ha & 0x04040404u, hb & 0x04040404u, ha & 0x08080808u, hb & 0x08080808u, bf[3][0], bf[3][1]);
}

// grid = (ceil(Lcap / SPAN), B*Hkv); SPAN = EST_STAGES * TS tokens per CTA.
template <int TS, bool INT_OUT, bool HAS_BIAS>
__global__ void __launch_bounds__(EST_THREADS)
estimate_kernel(const uint32_t* __restrict__ codes, const float* __restrict__ f_scale,
                const float* __restrict__ f_bias, const int32_t* __restrict__ n_indexed,
                const RbqQConst* __restrict__ qconst, int Hq, int Hkv, int Lcap, float sm_scale,
                float* __restrict__ scores, int32_t* __restrict__ dot_out, int32_t* __restrict__ pop_out) {
  constexpr int SPAN = EST_STAGES * TS;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint4* s_codes = reinterpret_cast<uint4*>(smem_raw);                           // [SPAN]
  float* s_fs = reinterpret_cast<float*>(smem_raw + (size_t)SPAN * 16);           // [SPAN]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)SPAN * 20);    // [EST_STAGES]

  const int bg = blockIdx.y, b = bg / Hkv, gk = bg % Hkv, G = Hq / Hkv;
  const int n = n_indexed[b];
  const int t0 = blockIdx.x * SPAN;
  if (t0 >= n) return;
  const int cnt = min(SPAN, n - t0);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int s = 0; s < EST_STAGES; ++s) mbar_init(&s_bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const size_t tok0 = (size_t)bg * Lcap + t0;
    for (int s = 0; s < EST_STAGES; ++s) {
      const int c = min(TS, cnt - s * TS);
      if (c <= 0) break;
      const int c4 = (c + 3) & ~3;                         // f_scale bytes must be a multiple of 16
      mbar_expect_tx(&s_bar[s], (uint32_t)(c * 16 + c4 * 4));
      bulk_g2s(s_codes + s * TS, codes + (tok0 + (size_t)s * TS) * RBQ_WORDS, (uint32_t)(c * 16), &s_bar[s]);
      bulk_g2s(s_fs + s * TS, f_scale + tok0 + (size_t)s * TS, (uint32_t)(c4 * 4), &s_bar[s]);
    }
  }
  // per-warp constants: B fragments (8 regs) and this lane's head constants
  const RbqQConst* qc = qconst + bg;
  const int g = lane >> 2, t = lane & 3;
  uint32_t bf[4][2];
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    const uint2 v = *reinterpret_cast<const uint2*>(&qc->bfrag[s][lane][0]);
    bf[s][0] = v.x; bf[s][1] = v.y;
  }
  const bool head_ok = t < G;
  const int hsel = head_ok ? t : 0;
  const float cA = qc->cA[hsel], cB = qc->cB[hsel], cD = qc->cD[hsel];
  const int init_d = qc->init_d[hsel], init_p = qc->init_p;
  const size_t row = ((size_t)b * Hq + gk * G + hsel) * Lcap;
  const size_t prow = (size_t)bg * Lcap;
  __syncthreads();                                         // barrier inits visible to all waiters

  const uint32_t* s_words = reinterpret_cast<const uint32_t*>(s_codes);
  const int ngroups = (cnt + 31) >> 5;
  for (int gi = warp; gi < ngroups; gi += EST_THREADS / 32) {
    const int base = gi << 5;                              // token offset inside the span
    mbar_wait(&s_bar[base / TS], 0);
    // lane (g,t) holds word t of tokens base+g, +8, +16, +24 (conflict-free: 4*(base+g)+t)
    const uint32_t w0 = s_words[(base + g) * 4 + t];
    const uint32_t w1 = s_words[(base + g + 8) * 4 + t];
    const uint32_t w2 = s_words[(base + g + 16) * 4 + t];
    const uint32_t w3 = s_words[(base + g + 24) * 4 + t];
    int c0[4] = {init_d, init_p, init_d, init_p};
    int c1[4] = {init_d, init_p, init_d, init_p};
    tile_mma(c0, w0, w1, bf);
    tile_mma(c1, w2, w3, bf);
    const int acc_d[4] = {c0[0], c0[2], c1[0], c1[2]};
    const int acc_p[4] = {c0[1], c0[3], c1[1], c1[3]};
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int tl = base + g + 8 * r;
      if (tl < cnt && head_ok) {
        const int tok = t0 + tl;
        if (INT_OUT) {
          dot_out[row + tok] = (acc_d[r] - init_d) >> 3;
          if (t == 0) pop_out[prow + tok] = (acc_p[r] - init_p) >> 3;
        } else {
          const float fd = __fsub_rn(__int_as_float(acc_d[r]), 12582912.0f);
          const float fp = __fsub_rn(__int_as_float(acc_p[r]), 12582912.0f);
          const float ip = fmaf(cA, fd, __fmul_rn(cB, fp));
          float sc = fmaf(s_fs[tl], ip, cD);
          if (HAS_BIAS) sc = fmaf(sm_scale, f_bias[row + tok], sc);
          scores[row + tok] = sc;
        }
      }
    }
  }
}

template <int TS, bool INT_OUT, bool HAS_BIAS>
int launch_t(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, cudaStream_t s) {
  constexpr int SPAN = EST_STAGES * TS;
  const size_t smem = (size_t)SPAN * 20 + EST_STAGES * 8;
  auto kern = estimate_kernel<TS, INT_OUT, HAS_BIAS>;
  static bool attr_set = false;
  if (!attr_set) {
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_set = true;
  }
  dim3 grid((ctx->cfg.max_tokens + SPAN - 1) / SPAN, ctx->cfg.batch * ctx->cfg.n_kv_heads);
  const RbqQConst* qc = reinterpret_cast<const RbqQConst*>(static_cast<char*>(ctx->ws) + ctx->off_qconst);
  kern<<<grid, EST_THREADS, smem, s>>>(idx->codes, idx->f_scale, idx->f_bias, idx->n_indexed, qc, ctx->cfg.n_q_heads,
                                       ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, ctx->sm_scale, scores, dot, pop);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

}  // namespace

int rbq_launch_estimate(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, cudaStream_t s) {
  constexpr int TS = 512;
  if (dot) return launch_t<TS, true, false>(ctx, idx, scores, dot, pop, s);
  if (idx->f_bias && idx->c_q) return launch_t<TS, false, true>(ctx, idx, scores, dot, pop, s);
  return launch_t<TS, false, false>(ctx, idx, scores, dot, pop, s);
}
