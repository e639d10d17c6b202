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
// by S3.
//
// Streaming: no shared memory.  The 32-token groups of all (sequence, KV head) pairs form one flat
// list that is cut into equal contiguous ranges, one per WARP (grid = a multiple of the SM count);
// a warp keeps two groups of loads in flight.  MMA rows are mapped to tokens so that lane (g, t)
// ends up with head t's logits of tokens 4g..4g+3: one 16-byte coalesced store per lane and group.
//
// Templated on W = D/32 code words per token (D = 64, 128, 256; the bit <-> MMA-operand mapping is rbq_bfrag_dim).
//
// Measured alternatives (round 2, profiles/r02_estimator.md): a persistent one-CTA-per-SM variant that stages the code
// stream in a shared-memory ring with 1-D bulk copies (UBLKCP) and runs S3 inside the CTA was 10 us SLOWER per step: the
// inner loop is bound by the ALU pipe (36 LOP3/SHF per 32-token group at 2 clk each) plus the IMMA pipe (~11 clk per
// IMMA.16832 in this mix), not by HBM, and a 200 KB CTA cannot become resident under its predecessor as these small CTAs do.
//
// Integer results are exact.  Epilogue in fp32 without cancellation:
//   acc_d = 4*(2*dot - sum(qu)), acc_p = 4*(2*pop - D)   (exact ints: accumulators start at
//   0x4B400000 - 4*sum(qu) / - 4*D, so reinterpreting as float and subtracting 2^23+2^22 converts)
//   score = f_scale*(cA*acc_d + cB*acc_p) + cD [+ sm_scale*f_bias].
#include "rbq_common.cuh"

RBQ_PROBE_DECL(est_probe);

namespace {

constexpr int EST_THREADS = 256;
constexpr int EST_WARPS = EST_THREADS / 32;
constexpr int EST_MAX_B = 1024;               // sequences whose group prefix fits the shared table

__device__ __forceinline__ void imma_16832(int (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                           uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// first k-step of a tile: D = A*B + C with C = the (biased) start values, so no accumulator initialisation moves
__device__ __forceinline__ void imma_16832_first(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                 uint32_t b0, uint32_t b1, int cd, int cp) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%11,%10,%11};"
               : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "r"(cd), "r"(cp));
}

// what lane (g, t) holds of one token: the 32-bit value(s) x of rbq_bfrag_dim
template <int W> struct TokX { uint32_t x[W == 8 ? 2 : 1]; };

template <int W>
__device__ __forceinline__ TokX<W> load_tok(const uint32_t* __restrict__ p, int t) {   // p: the token's first code word
  TokX<W> r;
  if (W == 4) {
    r.x[0] = __ldg(p + t);
  } else if (W == 8) {
    const uint2 v = __ldg(reinterpret_cast<const uint2*>(p) + t);
    r.x[0] = v.x; r.x[W == 8 ? 1 : 0] = v.y;
  } else {
    const uint32_t v = (__ldg(p + (t >> 1)) >> (16 * (t & 1))) & 0xFFFFu;
    r.x[0] = v | ((v >> 1) << 16);
  }
  return r;
}

// One 16-token tile: rows g (token value a) and g + 8 (token value b) of this lane's quad column.
template <int W>
__device__ __forceinline__ void tile_mma(int (&c)[4], const TokX<W>& a, const TokX<W>& b, const uint32_t (&bf)[W][2], int cd, int cp) {
  if (W == 2) {
    const uint32_t wa = a.x[0], wb = b.x[0], ha = wa >> 4, hb = wb >> 4;
    imma_16832_first(c, wa & 0x01010101u, wb & 0x01010101u, wa & 0x04040404u, wb & 0x04040404u, bf[0][0], bf[0][1], cd, cp);
    imma_16832(c, ha & 0x01010101u, hb & 0x01010101u, ha & 0x04040404u, hb & 0x04040404u, bf[1][0], bf[1][1]);
  } else {
#pragma unroll
    for (int u = 0; u < (W == 8 ? 2 : 1); ++u) {
      const uint32_t wa = a.x[u], wb = b.x[u], ha = wa >> 4, hb = wb >> 4;
      if (u == 0)
        imma_16832_first(c, wa & 0x01010101u, wb & 0x01010101u, wa & 0x02020202u, wb & 0x02020202u, bf[0][0], bf[0][1], cd, cp);
      else
        imma_16832(c, wa & 0x01010101u, wb & 0x01010101u, wa & 0x02020202u, wb & 0x02020202u, bf[4 * u][0], bf[4 * u][1]);
      imma_16832(c, wa & 0x04040404u, wb & 0x04040404u, wa & 0x08080808u, wb & 0x08080808u, bf[4 * u + 1][0], bf[4 * u + 1][1]);
      imma_16832(c, ha & 0x01010101u, hb & 0x01010101u, ha & 0x02020202u, hb & 0x02020202u, bf[4 * u + 2][0], bf[4 * u + 2][1]);
      imma_16832(c, ha & 0x04040404u, hb & 0x04040404u, ha & 0x08080808u, hb & 0x08080808u, bf[4 * u + 3][0], bf[4 * u + 3][1]);
    }
  }
}

template <int W> struct GroupLoad {   // what lane (g, t) needs of one 32-token group
  TokX<W> w[4];               // its share of the code of tokens 4g .. 4g+3
  float4 fs;                  // f_scale of tokens 4g .. 4g+3
};

// grid = k * SMs CTAs of EST_WARPS warps.  Flat group index -> (sequence b, KV head, 32-token group).
// F16: the factors are stored as binary16 (rbq_config.factor_dtype; 2 + D/8 bytes per unit instead of 4 + D/8)
template <int W, bool INT_OUT, bool HAS_BIAS, bool F16>
__global__ void __launch_bounds__(EST_THREADS, W == 8 ? 2 : 3)
estimate_kernel(const uint32_t* __restrict__ codes, const void* __restrict__ f_scale,
                const float* __restrict__ f_bias, const int32_t* __restrict__ n_indexed,
                const RbqQConst* __restrict__ qconst, int B, int Hq, int Hkv, int Lcap, float sm_scale,
                float* __restrict__ scores, int32_t* __restrict__ dot_out, int32_t* __restrict__ pop_out,
                uint32_t* __restrict__ rowmax_key) {
  __shared__ int s_gstart[EST_MAX_B + 1];     // exclusive prefix over sequences of Hkv * ceil(n_b / 32)
  rbq_pdl_trigger();                            // the wait for S3 comes after the first code loads are in flight
  if (threadIdx.x == 0) RBQ_STAMP(est_probe, 0);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3, G = Hq / Hkv;
  if (tid == 0) {
    int run = 0;
    for (int b = 0; b < B; ++b) { s_gstart[b] = run; run += Hkv * ((max(0, n_indexed[b]) + 31) >> 5); }
    s_gstart[B] = run;
  }
  __syncthreads();
  const long long total = s_gstart[B];
  const long long nwarps = (long long)gridDim.x * EST_WARPS, wid = (long long)blockIdx.x * EST_WARPS + warp;
  long long gcur = total * wid / nwarps;
  const long long gend = total * (wid + 1) / nwarps;
  if (gcur >= gend) { rbq_pdl_wait(); return; }
  bool first_segment = true;
  int b = 0;
  {
    int lo = 0, hi = B - 1;                    // last b with s_gstart[b] <= gcur
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if ((long long)s_gstart[mid] <= gcur) lo = mid; else hi = mid - 1; }
    b = lo;
  }
  const bool head_ok = t < G;
  const int hsel = head_ok ? t : 0;

  while (gcur < gend) {
    // segment: groups of one (b, KV head) handled by this warp
    while ((long long)s_gstart[b + 1] <= gcur) ++b;
    const int n = n_indexed[b];
    const int gpb = (n + 31) >> 5;                              // groups per (b, KV head)
    const int rel = (int)(gcur - s_gstart[b]);
    const int gk = rel / gpb, g0 = rel % gpb;
    const int g1 = (int)min((long long)gpb, (long long)g0 + (gend - gcur));
    const int bg = b * Hkv + gk;
    const size_t prow = (size_t)bg * Lcap;
    // lane (g, t): word t of tokens 4g..4g+3 of a group and their factors.  A token run beyond the allocation
    // (Lcap % 32 != 0) is clamped to its last 4 tokens (never stored); groups beyond the segment are not loaded.
    const uint32_t* cbase = codes + prow * W;
    const float* fbase = reinterpret_cast<const float*>(f_scale) + prow;          // F16: see load_at
    const __half* hbase = reinterpret_cast<const __half*>(f_scale) + prow;
    const int tok_clamp = Lcap - 4;
    auto load_at = [&](int gi) -> GroupLoad<W> {
      const int tk = min(gi * 32 + 4 * g, tok_clamp);
      const uint32_t* p = cbase + (size_t)tk * W;
      GroupLoad<W> r;
#pragma unroll
      for (int k = 0; k < 4; ++k) r.w[k] = load_tok<W>(p + k * W, t);
      if (F16) {
        const uint2 hv = __ldg(reinterpret_cast<const uint2*>(hbase + tk));
        const float2 f01 = __half22float2(*reinterpret_cast<const __half2*>(&hv.x)), f23 = __half22float2(*reinterpret_cast<const __half2*>(&hv.y));
        r.fs = make_float4(f01.x, f01.y, f23.x, f23.y);
      } else {
        r.fs = __ldg(reinterpret_cast<const float4*>(fbase + tk));
      }
      return r;
    };
    // three groups of loads in flight per warp; codes and factors do not depend on S3, its constants do
    GroupLoad<W> l0 = load_at(g0), l1 = l0, l2 = l0;
    if (g0 + 1 < g1) l1 = load_at(g0 + 1);
    if (g0 + 2 < g1) l2 = load_at(g0 + 2);
    if (first_segment) { rbq_pdl_wait(); first_segment = false; if (tid == 0) RBQ_STAMP(est_probe, 1); }   // S3's query constants and zeroed row maxima
    const RbqQConst* qc = qconst + bg;
    uint32_t bf[W][2];
#pragma unroll
    for (int s = 0; s < W; ++s) {
      const uint2 v = *reinterpret_cast<const uint2*>(&qc->bfrag[s][lane][0]);
      bf[s][0] = v.x; bf[s][1] = v.y;
    }
    const float cA = qc->cA[hsel], cB = qc->cB[hsel], cD = qc->cD[hsel];
    const int init_d = qc->init_d[hsel], init_p = qc->init_p;
    const size_t row = ((size_t)b * Hq + gk * G + hsel) * Lcap;

    float smax = -INFINITY;                                     // running max of this lane's head over the segment
    auto process = [&](const GroupLoad<W>& cur, int gi) {
      // tile 0: rows g / g+8 = tokens 4g / 4g+1 ; tile 1: tokens 4g+2 / 4g+3
      int c0[4], c1[4];
      tile_mma<W>(c0, cur.w[0], cur.w[1], bf, init_d, init_p);
      tile_mma<W>(c1, cur.w[2], cur.w[3], bf, init_d, init_p);
      const int acc_d[4] = {c0[0], c0[2], c1[0], c1[2]};
      const int acc_p[4] = {c0[1], c0[3], c1[1], c1[3]};
      const int tok = gi * 32 + 4 * g;                          // first of this lane's 4 tokens
      if (head_ok && tok < n) {
        if (INT_OUT) {
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            if (tok + r < n) {
              dot_out[row + tok + r] = (acc_d[r] - init_d) >> 3;
              if (t == 0) pop_out[prow + tok + r] = (acc_p[r] - init_p) >> 3;
            }
          }
        } else {
          const float fsv[4] = {cur.fs.x, cur.fs.y, cur.fs.z, cur.fs.w};
          float sc[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float fd = __fsub_rn(__int_as_float(acc_d[r]), 12582912.0f);
            const float fp = __fsub_rn(__int_as_float(acc_p[r]), 12582912.0f);
            const float ip = fmaf(cA, fd, __fmul_rn(cB, fp));
            sc[r] = fmaf(fsv[r], ip, cD);
          }
          if (HAS_BIAS) {
#pragma unroll
            for (int r = 0; r < 4; ++r) if (tok + r < n) sc[r] = fmaf(sm_scale, f_bias[row + tok + r], sc[r]);
          }
          if (tok + 3 < n) {
            *reinterpret_cast<float4*>(scores + row + tok) = make_float4(sc[0], sc[1], sc[2], sc[3]);
            smax = fmaxf(fmaxf(smax, fmaxf(sc[0], sc[1])), fmaxf(sc[2], sc[3]));
          } else {
#pragma unroll
            for (int r = 0; r < 4; ++r) if (tok + r < n) { scores[row + tok + r] = sc[r]; smax = fmaxf(smax, sc[r]); }
          }
        }
      }
    };
    for (int gi = g0; gi < g1; gi += 3) {
      process(l0, gi);
      if (gi + 3 < g1) l0 = load_at(gi + 3);
      if (gi + 1 < g1) process(l1, gi + 1);
      if (gi + 4 < g1) l1 = load_at(gi + 4);
      if (gi + 2 < g1) process(l2, gi + 2);
      if (gi + 5 < g1) l2 = load_at(gi + 5);
    }
    if (!INT_OUT) {                                             // row maximum for S6 (keys pre-zeroed by S3)
      smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, 4));
      smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, 8));
      smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, 16));
      if (g == 0 && head_ok && smax > -INFINITY && rowmax_key != nullptr)
        atomicMax(&rowmax_key[(size_t)b * Hq + gk * G + t], rbq_fkey(__fadd_rn(smax, 0.0f)));
    }
    gcur += g1 - g0;
  }
  if (tid == 0) RBQ_STAMP(est_probe, 2);
}

template <int W, bool INT_OUT, bool HAS_BIAS, bool F16>
int launch_f(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, uint32_t* rowmax_key, cudaStream_t s) {
  if (ctx->cfg.batch > EST_MAX_B) RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "batch %d > %d", ctx->cfg.batch, EST_MAX_B);
  // upper bound of the work: every sequence full; 3 CTAs (24 warps) per SM, fewer when there is little work
  const long long max_groups = (long long)ctx->cfg.batch * ctx->cfg.n_kv_heads * ((ctx->cfg.max_tokens + 31) / 32);
  long long ctas = (max_groups + 2 * EST_WARPS - 1) / (2 * EST_WARPS);          // >= 2 groups per warp
  const long long cap = (long long)ctx->sm_count * (W == 8 ? 2 : 3);
  if (ctas > cap) ctas = cap;
  if (ctas < 1) ctas = 1;
  const RbqQConst* qc = reinterpret_cast<const RbqQConst*>(static_cast<char*>(ctx->ws) + ctx->off_qconst);
  RBQ_CUDA_OK(ctx, rbq_launch_pdl(estimate_kernel<W, INT_OUT, HAS_BIAS, F16>, dim3((unsigned)ctas), dim3(EST_THREADS), 0, s,
                                  (const uint32_t*)idx->codes, (const void*)idx->f_scale, (const float*)idx->f_bias,
                                  (const int32_t*)idx->n_indexed, qc, ctx->cfg.batch, ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads,
                                  ctx->cfg.max_tokens, ctx->sm_scale, scores, dot, pop, rowmax_key));
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

template <int W, bool INT_OUT, bool HAS_BIAS>
int launch_t(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, uint32_t* rowmax_key, cudaStream_t s) {
  if (ctx->cfg.factor_dtype == RBQ_F16) return launch_f<W, INT_OUT, HAS_BIAS, true>(ctx, idx, scores, dot, pop, rowmax_key, s);
  return launch_f<W, INT_OUT, HAS_BIAS, false>(ctx, idx, scores, dot, pop, rowmax_key, s);
}

template <int W>
int launch_w(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, uint32_t* rowmax_key, cudaStream_t s) {
  if (dot) return launch_t<W, true, false>(ctx, idx, scores, dot, pop, rowmax_key, s);
  if (idx->f_bias && idx->c_q) return launch_t<W, false, true>(ctx, idx, scores, dot, pop, rowmax_key, s);
  return launch_t<W, false, false>(ctx, idx, scores, dot, pop, rowmax_key, s);
}

}  // namespace

// S4/S5 with the query constants of the rbq_launch_query in front of it (chained by programmatic dependent launch).
// rowmax_key (or NULL): receives the order-preserving keys of the row maxima by atomicMax -- must be zero on entry.
int rbq_launch_estimate(rbq_ctx* ctx, const rbq_index* idx, float* scores, int32_t* dot, int32_t* pop, uint32_t* rowmax_key,
                        cudaStream_t s) {
  switch (ctx->cfg.head_dim) {
    case 64: return launch_w<2>(ctx, idx, scores, dot, pop, rowmax_key, s);
    case 256: return launch_w<8>(ctx, idx, scores, dot, pop, rowmax_key, s);
    default: return launch_w<4>(ctx, idx, scores, dot, pop, rowmax_key, s);
  }
}

int rbq_probe_copy_estimate(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, est_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}
