// rbq_encode_fast.cu -- S1 / S2 in RBQ_ENC_FAST mode: Alg.1 with the dense
// D x D rotation on the 5th-generation tensor cores (the "O(N_h L D^2)" term of L774).
//
// y = x P with x = fl32(k) - c_k.  x and P are split into bf16 hi + lo parts and the product is taken as
// x_hi P_hi + x_lo P_hi + x_hi P_lo with fp32 accumulation (the dropped x_lo P_lo term and the split roundings are
// ~2^-17 ||x|| per output).  Unlike RBQ_ENC_EXACT this does not reproduce the canonical fp32 order of DESIGN.md R1: a
// code bit may differ from the oracle's where |y_j| <= 1e-5 ||x||, f_scale within 1e-5 relative (guard band of
// SURVEY.md 8(c) C1, checked in tests/test_gpu_parity.py::test_encode_fast_guard_band).
//
// Kernel: one CTA per SM, tcgen05.mma.cta_group::1.kind::f16 with M = 128 tokens, N = 128 outputs, K = 16 per
// instruction, accumulators in TMEM (all 512 columns: 2 groups x 2 buffers x 128).  The CTA is two independent
// 8-warp pipelines ("groups") plus one MMA-issuing warp per group:
//   group warps : raw K rows (prefetched into registers one tile ahead) -> x -> x_hi / x_lo written to shared memory
//                 in the canonical K-major no-swizzle UMMA layout (8 x 16-byte core matrices; SBO = 128 B between
//                 8-row groups, LBO = 2080 B between 16-byte K chunks: 2048 + 32 so that the 16-byte operand stores
//                 of a quarter-warp hit 8 different bank groups) -> mbarrier "full";
//                 then the epilogue of the previous tile: tcgen05.ld (one token row per thread, 64 columns per warp),
//                 l1 and sign bits, the two column halves meet in shared memory, codes / f_scale stored coalesced.
//   issuer warp : waits "full", one lane issues the 24 MMAs of the tile, tcgen05.commit -> mbarrier "done".
// P_hi / P_lo are staged once per CTA in the same layout (B operand, N x K); for the Walsh-Hadamard rotation the dense
// matrix diag(s) H / sqrt(D) is generated in that loop from the sign vector (the same kernel serves both rotations).  MMA(t + 1) runs under epilogue(t) and
// under the other group's operand build.
#include "rbq_common.cuh"

namespace {

__device__ __forceinline__ uint32_t ef_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// (v0, v1) -> packed bf16 hi parts and packed bf16 lo parts (lo = bf16(v - hi))
__device__ __forceinline__ void ef_split(float v0, float v1, uint32_t& hi, uint32_t& lo) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  const __nv_bfloat162 l = __floats2bfloat162_rn(v0 - rbq_bf16lo(hi), v1 - rbq_bf16hi(hi));
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

constexpr int T5_GROUPS = 2;                                 // independent 8-warp pipelines per CTA (tile t of group g overlaps tile t' of the other)
constexpr int T5_GTHREADS = 256;
constexpr int T5_THREADS = T5_GROUPS * T5_GTHREADS + T5_GROUPS * 32;   // + one MMA-issuing warp per group
constexpr int T5_TOK = 128;
constexpr int T5_LBO = 2048 + 32;                            // bytes between K chunks (8 elements) of an operand tile
constexpr int T5_SBO = 128;                                  // bytes between 8-row groups
constexpr int T5_TILE = 16 * T5_LBO;                         // one 128 x 128 bf16 operand tile
constexpr int T5_SMEM = (2 + 2 * T5_GROUPS) * T5_TILE + RBQ_D * 4 + T5_GROUPS * (2 * T5_TOK * 4 + 2 * T5_TOK * 16) + 64;   // B_hi B_lo | per group A_hi A_lo | c_k | per group n2 x 2, exchange x 2 (tile parity) | misc
constexpr uint32_t T5_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(RBQ_D >> 3) << 17) | ((uint32_t)(T5_TOK >> 4) << 24);

__device__ __forceinline__ uint64_t t5_desc(uint32_t smem_addr) {
  return (uint64_t)((smem_addr >> 4) & 0x3FFFu) | ((uint64_t)(T5_LBO >> 4) << 16) | ((uint64_t)(T5_SBO >> 4) << 32) | (1ull << 46);
}
__device__ __forceinline__ void t5_mma(uint32_t tmem_d, uint64_t a_desc, uint64_t b_desc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d), "l"(a_desc), "l"(b_desc), "r"(T5_IDESC), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void t5_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,"
      "%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
        "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void t5_group_sync(int grp) { asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(T5_GTHREADS) : "memory"); }
// 8 consecutive floats -> packed bf16 hi parts and lo parts (16 bytes each)
__device__ __forceinline__ void t5_split8(const float (&v)[8], uint4& hi, uint4& lo) {
  ef_split(v[0], v[1], hi.x, lo.x); ef_split(v[2], v[3], hi.y, lo.y);
  ef_split(v[4], v[5], hi.z, lo.z); ef_split(v[6], v[7], hi.w, lo.w);
}

__global__ void __launch_bounds__(T5_THREADS, 1)
encode_tc5_kernel(const __nv_bfloat16* __restrict__ K, long long sb, long long sh, long long st,
                  const int32_t* __restrict__ t_begin, const int32_t* __restrict__ t_count, int fixed_count, int Hkv,
                  int Lcap, const float* __restrict__ rot, int wh, const float* __restrict__ c_k, uint32_t* __restrict__ codes,
                  void* __restrict__ f_scale, int fs_f16) {
  extern __shared__ __align__(128) unsigned char t5_smem[];
  const bool issuer = threadIdx.x >= T5_GROUPS * T5_GTHREADS;  // the last T5_GROUPS warps only issue MMAs
  const int grp = issuer ? ((int)threadIdx.x - T5_GROUPS * T5_GTHREADS) >> 5 : (int)threadIdx.x / T5_GTHREADS;   // pipeline group
  unsigned char* s_bh = t5_smem;
  unsigned char* s_bl = t5_smem + T5_TILE;
  unsigned char* s_ah = t5_smem + (2 + 2 * grp) * T5_TILE;
  unsigned char* s_al = s_ah + T5_TILE;
  float* s_ck = reinterpret_cast<float*>(t5_smem + (2 + 2 * T5_GROUPS) * T5_TILE);
  float* s_n2 = s_ck + RBQ_D + grp * 2 * T5_TOK;                // two buffers (tile parity)
  // per row: {l1 bits, word 2, word 3, -} of the upper column half; two buffers (tile parity), so that the hc == 1 warps of
  // tile t + 1 never overwrite what a slow hc == 0 warp of tile t has not read yet (one group barrier per tile)
  uint4* s_ex = reinterpret_cast<uint4*>(s_ck + RBQ_D + T5_GROUPS * 2 * T5_TOK) + grp * 2 * T5_TOK;
  uint64_t* s_bar0 = reinterpret_cast<uint64_t*>(reinterpret_cast<uint4*>(s_ck + RBQ_D + T5_GROUPS * 2 * T5_TOK) + T5_GROUPS * 2 * T5_TOK);
  uint64_t* s_bar = s_bar0 + grp;                             // accumulator ready (tcgen05.commit)
  uint64_t* s_full = s_bar0 + T5_GROUPS + grp;                // A operands written (all threads of the group arrive)
  uint32_t* s_tmem = reinterpret_cast<uint32_t*>(s_bar0 + 2 * T5_GROUPS);

  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int tb = t_begin ? t_begin[b] : 0;
  const int cnt = min(t_count ? t_count[b] : fixed_count, Lcap - tb);   // never past the capacity (append overflow, rbq_status_flags)
  if ((int)blockIdx.x * T5_GROUPS * T5_TOK >= cnt) return;
  const int tid = threadIdx.x % T5_GTHREADS, warp = tid >> 5, lane = tid & 31;   // indices inside the group

  if (threadIdx.x < 32) {                                     // TMEM: 128 columns x 128 lanes of fp32 accumulator per group
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(ef_smem_u32(s_tmem)), "r"((uint32_t)(256 * T5_GROUPS)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 32) {
    for (int i = 0; i < T5_GROUPS; ++i) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ef_smem_u32(s_bar0 + i)) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ef_smem_u32(s_bar0 + T5_GROUPS + i)), "r"(T5_GTHREADS) : "memory");
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // B operands: B[n = j][k = i] = P[i][j], hi / lo parts; two consecutive k per store
  for (int e = threadIdx.x; e < RBQ_D * RBQ_D / 2; e += T5_THREADS) {
    const int j = e & 127, i2 = (e >> 7) * 2;
    uint32_t hi, lo;
    float p0, p1;
    if (wh) {                                                   // Walsh-Hadamard: P = diag(s) H / sqrt(D), H_ij = (-1)^popc(i & j)
      const float r = 1.0f / sqrtf((float)RBQ_D);
      p0 = __ldg(rot + i2) * ((__popc(i2 & j) & 1) ? -r : r);
      p1 = __ldg(rot + i2 + 1) * ((__popc((i2 + 1) & j) & 1) ? -r : r);
    } else {
      p0 = __ldg(rot + i2 * RBQ_D + j);
      p1 = __ldg(rot + (i2 + 1) * RBQ_D + j);
    }
    ef_split(p0, p1, hi, lo);
    const int off = (i2 >> 3) * T5_LBO + (j >> 3) * T5_SBO + (j & 7) * 16 + (i2 & 7) * 2;
    *reinterpret_cast<uint32_t*>(s_bh + off) = hi;
    *reinterpret_cast<uint32_t*>(s_bl + off) = lo;
  }
  if (threadIdx.x < RBQ_D) s_ck[threadIdx.x] = c_k[(size_t)bg * RBQ_D + threadIdx.x];
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *s_tmem, tmem = tmem_base + (uint32_t)(256 * grp);   // two 128-column accumulators per group

  const __nv_bfloat16* base = K + (long long)b * sb + (long long)g * sh + (long long)tb * st;
  uint32_t phase = 0;
  const int stride = (int)gridDim.x * T5_GROUPS * T5_TOK;
  const int r8 = lane >> 2, c4 = lane & 3;
  uint4 kr[8];                                                // raw K pieces of the tile being staged: [row half][chunk group]

  // raw K of tile `tile0` -> registers (thread item = (row, 8-column chunk); a warp covers 8 rows x 4 chunks per step)
  auto load_tile = [&](int tile0) {
    const int ntok = min(T5_TOK, cnt - tile0);
#pragma unroll
    for (int hr = 0; hr < 2; ++hr) {
      const int r = 64 * hr + 8 * warp + r8;
#pragma unroll
      for (int cgp = 0; cgp < 4; ++cgp)
        kr[hr * 4 + cgp] = (r < ntok) ? __ldg(reinterpret_cast<const uint4*>(base + (long long)(tile0 + r) * st + (4 * cgp + c4) * 8))
                                      : make_uint4(0u, 0u, 0u, 0u);
    }
  };
  // registers -> A operands x = k - c_k (hi / lo) and ||x||^2 per row
  // (rows past the end of the sequence hold -c_k: their accumulator rows are never stored)
  auto build_a = [&](float* n2buf) {
#pragma unroll
    for (int hr = 0; hr < 2; ++hr) {
      const int r = 64 * hr + 8 * warp + r8;
      float n2 = 0.0f;
#pragma unroll
      for (int cgp = 0; cgp < 4; ++cgp) {
        const int c = 4 * cgp + c4;
        const uint4 u = kr[hr * 4 + cgp];
        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
        const float4 ca = *reinterpret_cast<const float4*>(s_ck + c * 8), cb = *reinterpret_cast<const float4*>(s_ck + c * 8 + 4);
        float x[8];
        x[0] = rbq_bf16lo(w[0]) - ca.x; x[1] = rbq_bf16hi(w[0]) - ca.y; x[2] = rbq_bf16lo(w[1]) - ca.z; x[3] = rbq_bf16hi(w[1]) - ca.w;
        x[4] = rbq_bf16lo(w[2]) - cb.x; x[5] = rbq_bf16hi(w[2]) - cb.y; x[6] = rbq_bf16lo(w[3]) - cb.z; x[7] = rbq_bf16hi(w[3]) - cb.w;
#pragma unroll
        for (int k = 0; k < 8; ++k) n2 = fmaf(x[k], x[k], n2);
        uint4 hi, lo;
        t5_split8(x, hi, lo);
        const int off = c * T5_LBO + (r >> 3) * T5_SBO + (r & 7) * 16;
        *reinterpret_cast<uint4*>(s_ah + off) = hi;
        *reinterpret_cast<uint4*>(s_al + off) = lo;
      }
      n2 += __shfl_xor_sync(0xffffffffu, n2, 1);
      n2 += __shfl_xor_sync(0xffffffffu, n2, 2);
      if (c4 == 0) n2buf[r] = n2;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy operand stores -> async proxy (tensor core)
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(ef_smem_u32(s_full)) : "memory");
  };
  // 24 MMAs by one thread: x_hi P_hi (8 k-steps), x_lo P_hi, x_hi P_lo, into accumulator buffer `buf`
  auto issue = [&](int buf) {
    if (lane == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t d = tmem + (uint32_t)(128 * buf);
      const uint32_t ah = ef_smem_u32(s_ah), al = ef_smem_u32(s_al), bh = ef_smem_u32(s_bh), bl = ef_smem_u32(s_bl);
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) t5_mma(d, t5_desc(ah + ks * 2 * T5_LBO), t5_desc(bh + ks * 2 * T5_LBO), ks > 0 ? 1u : 0u);
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) t5_mma(d, t5_desc(al + ks * 2 * T5_LBO), t5_desc(bh + ks * 2 * T5_LBO), 1u);
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) t5_mma(d, t5_desc(ah + ks * 2 * T5_LBO), t5_desc(bl + ks * 2 * T5_LBO), 1u);
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(ef_smem_u32(s_bar)) : "memory");
    }
  };
  // accumulator buffer `buf` -> codes and f_scale: thread = token row 32 (warp & 3) + lane, columns 64 (warp >> 2) .. + 63
  auto epilogue = [&](int tile0, int buf, const float* n2buf) {
    const int ntok = min(T5_TOK, cnt - tile0);
    const int q = warp & 3, hc = warp >> 2, r = 32 * q + lane;
    const uint32_t ta = tmem + (uint32_t)(128 * buf) + ((uint32_t)(32 * q) << 16) + (uint32_t)(64 * hc);
    float l1 = 0.0f;
    uint32_t w0 = 0u, w1 = 0u;
    uint32_t y[32];
    // code bit j = 1 - sign bit of y_j, shifted in from j = 31 down (one funnel shift per element).  y_j = +0 gives a 1
    // where "y_j > 0" gives 0: inside the guard band, and rows with x = 0 (l1 = 0) are forced to zero codes below.
    t5_ld32(ta, y);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int j = 31; j >= 0; --j) { l1 += fabsf(__uint_as_float(y[j])); w0 = __funnelshift_l(y[j], w0, 1); }
    t5_ld32(ta + 32u, y);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
#pragma unroll
    for (int j = 31; j >= 0; --j) { l1 += fabsf(__uint_as_float(y[j])); w1 = __funnelshift_l(y[j], w1, 1); }
    w0 = ~w0;
    w1 = ~w1;
    uint4* ex_buf = s_ex + buf * T5_TOK;
    if (hc == 1) ex_buf[r] = make_uint4(__float_as_uint(l1), w0, w1, 0u);
    t5_group_sync(grp);
    if (hc == 0 && r < ntok) {
      const uint4 ex = ex_buf[r];
      const float l1t = l1 + __uint_as_float(ex.x);
      const size_t tok = (size_t)bg * Lcap + tb + tile0 + r;
      const bool zero = l1t == 0.0f;
      reinterpret_cast<uint4*>(codes)[tok] = zero ? make_uint4(0u, 0u, 0u, 0u) : make_uint4(w0, w1, ex.y, ex.z);
      rbq_store_factor(f_scale, fs_f16, tok, zero ? 0.0f : n2buf[r] / l1t);
    }
  };

  // bounded spin on an mbarrier phase: a descriptor mistake must trap, not hang the GPU
  auto wait_bar = [&](uint64_t* bar, uint32_t ph) {
    uint32_t done = 0;
    for (uint32_t spin = 0; !done; ++spin) {
      asm volatile(
          "{\n\t"
          ".reg .pred p;\n\t"
          "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
          "selp.u32 %0, 1, 0, p;\n\t"
          "}\n" : "=r"(done) : "r"(ef_smem_u32(bar)), "r"(ph) : "memory");
      if (spin > (1u << 24)) __trap();
    }
  };
  // Per group: MMA(t + 1) runs under epilogue(t); the raw K of tile t + 1 is in flight while MMA(t) is awaited.
  int t = ((int)blockIdx.x * T5_GROUPS + grp) * T5_TOK;
  if (issuer) {
    for (int it = 0; t < cnt; t += stride, ++it) {
      wait_bar(s_full, phase);
      phase ^= 1u;
      issue(it & 1);
      __syncwarp();
    }
  } else {
    if (t < cnt) {
      load_tile(t);
      build_a(s_n2);
      if (t + stride < cnt) load_tile(t + stride);
    }
    for (int it = 0; t < cnt; ++it) {
      const int tn = t + stride;
      wait_bar(s_bar, phase);
      phase ^= 1u;
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      if (tn < cnt) {
        build_a(s_n2 + ((it + 1) & 1) * T5_TOK);                // tile tn (its raw K was loaded one epilogue ago)
        if (tn + stride < cnt) load_tile(tn + stride);          // in flight during the epilogue below
      }
      epilogue(t, it & 1, s_n2 + (it & 1) * T5_TOK);
      t = tn;
    }
  }
  __syncthreads();
  if (threadIdx.x < 32)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)(256 * T5_GROUPS)) : "memory");
}

}  // namespace

int rbq_launch_encode_fast(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count, int fixed_count,
                           int max_count, const rbq_index* idx, cudaStream_t s) {
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_ENC_FAST, encode_tc5_kernel, T5_SMEM);
  const int BG = ctx->cfg.batch * ctx->cfg.n_kv_heads;
  const int tiles = (max_count + T5_GROUPS * T5_TOK - 1) / (T5_GROUPS * T5_TOK);
  int gx = ctx->sm_count / BG;                                // one CTA per SM, a single wave; each CTA loops over its tiles
  gx = gx < 1 ? 1 : (gx > tiles ? tiles : gx);
  encode_tc5_kernel<<<dim3(gx, BG), T5_THREADS, T5_SMEM, s>>>((const __nv_bfloat16*)kv.k, kv.sb, kv.sh, kv.st, t_begin, t_count,
                                                             fixed_count, ctx->cfg.n_kv_heads, ctx->cfg.max_tokens,
                                                             ctx->cfg.rot, ctx->cfg.rot_kind == RBQ_ROT_WH ? 1 : 0, idx->c_k,
                                                             idx->codes, idx->f_scale, ctx->cfg.factor_dtype == RBQ_F16 ? 1 : 0);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
