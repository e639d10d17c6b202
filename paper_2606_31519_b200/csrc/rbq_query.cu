// rbq_query.cu -- S3: query pre-processing and INT4 quantisation
// (Alg.2 lines 4-6, L168-172; Eq.5; L524; readings R5/R6/R12 of DESIGN.md).
//
//   xq = q - c_q ; qn = ||xq||_2 ; u = xq/qn ; q' = u P (canonical fp32 order, as S1) ;
//   q_l = min q', q_r = max q', Delta = (q_r - q_l)/15 ; qu_j = clamp(floor((q'_j-q_l)/Delta + 1/2), 0, 15).
// One CTA per (sequence, KV head), one 128-thread slice per query head of the group.  Besides the
// optional public outputs (qu, qparams) it writes the private RbqQConst block: the u8 B-operand
// fragments of the estimator MMA and the per-head reconstruction constants of Eq.20 / Eq.2.
#include "rbq_common.cuh"

namespace {

template <typename TQ>
__global__ void __launch_bounds__(RBQ_MAX_G * RBQ_D)
query_kernel(const TQ* __restrict__ q, const float* __restrict__ c_q, const float* __restrict__ c_k,
             const float* __restrict__ rot, int rot_kind, int Hq, int Hkv, float sm_scale,
             uint8_t* __restrict__ qu_out, float* __restrict__ qparams, RbqQConst* __restrict__ qc_out,
             uint32_t* __restrict__ rowmax_key, TQ* __restrict__ q_copy) {
  rbq_pdl_trigger();                               // S4/S5 may become resident while this kernel runs
  const int G = Hq / Hkv;
  const int bg = blockIdx.x, b = bg / Hkv, g = bg % Hkv;
  const int hs = threadIdx.x >> 7, j = threadIdx.x & 127;      // head slice, dim
  const int h = g * G + min(hs, G - 1);              // slices beyond G recompute head G-1, write nothing
  const size_t row = (size_t)b * Hq + h;

  extern __shared__ __align__(16) float s_rot[];  // dense: P [D][D] staged with one round of independent 128-bit loads
  __shared__ float s_ck[RBQ_D], s_cq[RBQ_MAX_G][RBQ_D];
  __shared__ __align__(16) float s_x[RBQ_MAX_G][RBQ_D];      // xq, then u
  __shared__ float s_y[RBQ_MAX_G][RBQ_D];      // q'
  __shared__ float s_red[RBQ_MAX_G][8];        // per-warp min / max
  __shared__ int s_isum[RBQ_MAX_G][4];
  __shared__ float s_qn[RBQ_MAX_G];
  __shared__ double s_dot[RBQ_MAX_G][2];
  __shared__ __align__(8) unsigned long long s_bar;
  __shared__ double s_dred[RBQ_MAX_G][2][4];
  __shared__ uint8_t s_qu[RBQ_MAX_G][RBQ_D];

  const float qv = rbq_ld_elem(q, row * RBQ_D + j);
  if (q_copy != nullptr && hs < G) q_copy[row * RBQ_D + j] = q[row * RBQ_D + j];   // q in mapped host memory: device copy for S7
  const float cqv = c_q ? c_q[row * RBQ_D + j] : 0.0f;
  const float ckv = c_k[(size_t)bg * RBQ_D + j];
  if (rot_kind == RBQ_ROT_DENSE && threadIdx.x == 0) {   // P -> shared memory by ONE bulk copy (TMA); awaited just before the rotation
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)(RBQ_D * RBQ_D * 4)) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     (uint32_t)__cvta_generic_to_shared(s_rot)), "l"(rot), "r"((uint32_t)(RBQ_D * RBQ_D * 4)), "r"(bar) : "memory");
  }
  const float xq = c_q ? __fsub_rn(qv, cqv) : qv;
  s_x[hs][j] = xq;
  s_y[hs][j] = qv;                               // staged for the fp64 dot chains below
  s_cq[hs][j] = cqv;
  if (hs == 0) s_ck[j] = ckv;
  __syncthreads();
  // ||xq||: the canonical sequential fp32 chain (R1) on one thread per head; the two fp64 dot products
  // <q,c_k>, <c_q,c_k> (exact products, fp64 sums, rounded to fp32 at the end) as a fixed reduction tree.
  {
    double p0 = (double)qv * (double)ckv;
    double p1 = c_q ? (double)cqv * (double)ckv : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      p0 += __shfl_xor_sync(0xffffffffu, p0, o);
      p1 += __shfl_xor_sync(0xffffffffu, p1, o);
    }
    if ((j & 31) == 0) { s_dred[hs][0][j >> 5] = p0; s_dred[hs][1][j >> 5] = p1; }
  }
  if (j == 0) {
    // compact loops on purpose: this code runs once per launch, so straight-line code is instruction-fetch bound
    float n2 = 0.0f;
#pragma unroll 1
    for (int i0 = 0; i0 < RBQ_D; i0 += 16) {
      float4 xv[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) xv[k] = *reinterpret_cast<const float4*>(&s_x[hs][i0 + 4 * k]);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        n2 = fmaf(xv[k].x, xv[k].x, n2); n2 = fmaf(xv[k].y, xv[k].y, n2);
        n2 = fmaf(xv[k].z, xv[k].z, n2); n2 = fmaf(xv[k].w, xv[k].w, n2);
      }
    }
    s_qn[hs] = __fsqrt_rn(n2);
  }
  __syncthreads();
  if (j == 0) {
    s_dot[hs][0] = (s_dred[hs][0][0] + s_dred[hs][0][1]) + (s_dred[hs][0][2] + s_dred[hs][0][3]);
    s_dot[hs][1] = (s_dred[hs][1][0] + s_dred[hs][1][1]) + (s_dred[hs][1][2] + s_dred[hs][1][3]);
  }
  const float qn = s_qn[hs];
  const float u = (qn > 0.0f) ? __fdiv_rn(xq, qn) : 0.0f;
  s_x[hs][j] = u;
  __syncthreads();
  if (rot_kind == RBQ_ROT_DENSE) {                 // P has landed (the barrier above also made the mbarrier init visible)
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n"
        "@p bra LAB_DONE_%=;\n"
        "bra LAB_WAIT_%=;\n"
        "LAB_DONE_%=:\n"
        "}\n" ::"r"(bar) : "memory");
  }

  float qp;
  if (rot_kind == RBQ_ROT_DENSE) {
    // Threads 0..255: one output column for TWO heads of the group each: one shared-memory read of P[i][j] feeds two
    // independent canonical chains (one read per head would be bound by shared-memory bandwidth, one read for all
    // four heads by the FMA issue rate of four warps).
    if (threadIdx.x < 2 * RBQ_D) {
      const int jj = threadIdx.x & (RBQ_D - 1), hp = (threadIdx.x >> 7) * 2;
      float a0 = 0.0f, a1 = 0.0f;
#pragma unroll 2
      for (int i0 = 0; i0 < RBQ_D; i0 += 8) {
        float rv[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) rv[k] = s_rot[(i0 + k) * RBQ_D + jj];
        const float4 xa = *reinterpret_cast<const float4*>(&s_x[hp][i0]), xb = *reinterpret_cast<const float4*>(&s_x[hp][i0 + 4]);
        const float4 ya = *reinterpret_cast<const float4*>(&s_x[hp + 1][i0]), yb = *reinterpret_cast<const float4*>(&s_x[hp + 1][i0 + 4]);
        a0 = fmaf(xa.x, rv[0], a0); a1 = fmaf(ya.x, rv[0], a1);
        a0 = fmaf(xa.y, rv[1], a0); a1 = fmaf(ya.y, rv[1], a1);
        a0 = fmaf(xa.z, rv[2], a0); a1 = fmaf(ya.z, rv[2], a1);
        a0 = fmaf(xa.w, rv[3], a0); a1 = fmaf(ya.w, rv[3], a1);
        a0 = fmaf(xb.x, rv[4], a0); a1 = fmaf(yb.x, rv[4], a1);
        a0 = fmaf(xb.y, rv[5], a0); a1 = fmaf(yb.y, rv[5], a1);
        a0 = fmaf(xb.z, rv[6], a0); a1 = fmaf(yb.z, rv[6], a1);
        a0 = fmaf(xb.w, rv[7], a0); a1 = fmaf(yb.w, rv[7], a1);
      }
      s_y[hp][jj] = a0; s_y[hp + 1][jj] = a1;
    }
    __syncthreads();
    qp = s_y[hs][j];
  } else {
    // warp 0 of the slice runs the 128-point butterflies (4 elements per lane), as in S1
    if (j < 32) {
      const int lane = j;
      float u0 = __fmul_rn(rot[lane * 4 + 0], s_x[hs][lane * 4 + 0]);
      float u1 = __fmul_rn(rot[lane * 4 + 1], s_x[hs][lane * 4 + 1]);
      float u2 = __fmul_rn(rot[lane * 4 + 2], s_x[hs][lane * 4 + 2]);
      float u3 = __fmul_rn(rot[lane * 4 + 3], s_x[hs][lane * 4 + 3]);
      float a, c;
      a = __fadd_rn(u0, u1); c = __fsub_rn(u0, u1); u0 = a; u1 = c;
      a = __fadd_rn(u2, u3); c = __fsub_rn(u2, u3); u2 = a; u3 = c;
      a = __fadd_rn(u0, u2); c = __fsub_rn(u0, u2); u0 = a; u2 = c;
      a = __fadd_rn(u1, u3); c = __fsub_rn(u1, u3); u1 = a; u3 = c;
#pragma unroll
      for (int m = 1; m < 32; m <<= 1) {
        const bool up = (lane & m) != 0;
        float p0 = __shfl_xor_sync(0xffffffffu, u0, m), p1 = __shfl_xor_sync(0xffffffffu, u1, m);
        float p2 = __shfl_xor_sync(0xffffffffu, u2, m), p3 = __shfl_xor_sync(0xffffffffu, u3, m);
        u0 = up ? __fsub_rn(p0, u0) : __fadd_rn(u0, p0);
        u1 = up ? __fsub_rn(p1, u1) : __fadd_rn(u1, p1);
        u2 = up ? __fsub_rn(p2, u2) : __fadd_rn(u2, p2);
        u3 = up ? __fsub_rn(p3, u3) : __fadd_rn(u3, p3);
      }
      const float c1 = (float)(1.0 / sqrt((double)RBQ_D));
      s_y[hs][lane * 4 + 0] = __fmul_rn(u0, c1);
      s_y[hs][lane * 4 + 1] = __fmul_rn(u1, c1);
      s_y[hs][lane * 4 + 2] = __fmul_rn(u2, c1);
      s_y[hs][lane * 4 + 3] = __fmul_rn(u3, c1);
    }
    __syncthreads();
    qp = s_y[hs][j];
  }

  // min / max over the 128 dims of the slice
  float mn = qp, mx = qp;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  }
  const int wslice = (j >> 5);
  if ((j & 31) == 0) { s_red[hs][wslice] = mn; s_red[hs][4 + wslice] = mx; }
  __syncthreads();
  const float ql = fminf(fminf(s_red[hs][0], s_red[hs][1]), fminf(s_red[hs][2], s_red[hs][3]));
  const float qr = fmaxf(fmaxf(s_red[hs][4], s_red[hs][5]), fmaxf(s_red[hs][6], s_red[hs][7]));
  const float delta = __fdiv_rn(__fsub_rn(qr, ql), 15.0f);
  int v = 0;
  if (delta > 0.0f) {
    const float t = __fdiv_rn(__fsub_rn(qp, ql), delta);
    v = (int)floorf(__fadd_rn(t, 0.5f));
    v = min(15, max(0, v));
  }
  s_qu[hs][j] = (uint8_t)v;
  int sv = v;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sv += __shfl_xor_sync(0xffffffffu, sv, o);
  if ((j & 31) == 0) s_isum[hs][wslice] = sv;
  __syncthreads();
  const int sumq = s_isum[hs][0] + s_isum[hs][1] + s_isum[hs][2] + s_isum[hs][3];

  if (hs < G && j == 0) rowmax_key[row] = 0u;                  // S5 accumulates the row maximum with atomicMax
  if (hs < G) {
    if (qu_out) qu_out[row * RBQ_D + j] = (uint8_t)v;
    if (j == 0) {
      const float q_ck = (float)s_dot[hs][0], cq_ck = (float)s_dot[hs][1];
      if (qparams) {
        float* o = qparams + row * 6;
        o[0] = qn; o[1] = ql; o[2] = delta; o[3] = (float)sumq; o[4] = q_ck; o[5] = cq_ck;
      }
      RbqQConst* qc = qc_out + bg;
      qc->cA[hs] = (float)((double)sm_scale * (double)qn * (double)delta * 0.25);
      qc->cB[hs] = (float)((double)sm_scale * (double)qn * (double)ql * 0.25);
      qc->cD[hs] = (float)((double)sm_scale * ((double)q_ck - (double)cq_ck));
      qc->init_d[hs] = 0x4B400000 - 4 * sumq;
      if (hs == 0) qc->init_p = 0x4B400000 - 4 * RBQ_D;
    }
  }
  // B-operand fragments: word (s, lane, r): byte i <-> k = 4*t' + i (+16 for r = 1), column n = g'
  //   dim = 32*t' + 8*i + 2*s + r, value = (n odd ? 1 : qu[head n/2][dim]) << (3 - ((2*s + r) & 3))
  if (threadIdx.x < 256) {
    const int w = threadIdx.x, s = w >> 6, lane = (w >> 1) & 31, r = w & 1;
    const int gp = lane >> 2, tp = lane & 3;
    const int e = 2 * s + r, sh = 3 - (e & 3);
    uint32_t word = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int dim = 32 * tp + 8 * i + e;
      uint32_t val = 0;
      if (gp & 1) val = ((gp >> 1) < G) ? 1u : 0u;
      else if ((gp >> 1) < G) val = s_qu[gp >> 1][dim];
      word |= (val << sh) << (8 * i);
    }
    qc_out[bg].bfrag[s][lane][r] = word;
  }
}

}  // namespace

int rbq_launch_query(rbq_ctx* ctx, const void* q, const rbq_index* idx, uint8_t* qu, float* qparams, void* q_copy, cudaStream_t s) {
  const int BG = ctx->cfg.batch * ctx->cfg.n_kv_heads;
  RbqQConst* qc = reinterpret_cast<RbqQConst*>(static_cast<char*>(ctx->ws) + ctx->off_qconst);
  uint32_t* rk = reinterpret_cast<uint32_t*>(static_cast<char*>(ctx->ws) + ctx->off_rowmax);
  const int threads = max(256, ctx->G * RBQ_D);
  const size_t smem = ctx->cfg.rot_kind == RBQ_ROT_DENSE ? (size_t)RBQ_D * RBQ_D * sizeof(float) : 0;
  if (!(ctx->attr_mask & RBQ_ATTR_QUERY)) {
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(query_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, RBQ_D * RBQ_D * 4));
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(query_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, RBQ_D * RBQ_D * 4));
    ctx->attr_mask |= RBQ_ATTR_QUERY;
  }
  if (ctx->cfg.q_dtype == RBQ_BF16)
    query_kernel<<<BG, threads, smem, s>>>((const __nv_bfloat16*)q, idx->c_q, idx->c_k, ctx->cfg.rot, ctx->cfg.rot_kind,
                                           ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads, ctx->sm_scale, qu, qparams, qc, rk, (__nv_bfloat16*)q_copy);
  else
    query_kernel<<<BG, threads, smem, s>>>((const float*)q, idx->c_q, idx->c_k, ctx->cfg.rot, ctx->cfg.rot_kind,
                                           ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads, ctx->sm_scale, qu, qparams, qc, rk, (float*)q_copy);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
