// rbq_encode_fast.cu -- S1 / S2 in RBQ_ENC_FAST mode: Alg.1 with the dense
// D x D rotation on the tensor pipe (the "O(N_h L D^2)" term of L774).
//
// y = x P with x = fl32(k) - c_k.  x and P are split into bf16 hi + lo parts and the product is taken as
// x_hi P_hi + x_lo P_hi + x_hi P_lo with mma.sync.m16n8k16.bf16 and fp32 accumulation (the dropped x_lo P_lo term and
// the split roundings are ~2^-17 ||x|| per output).  Unlike RBQ_ENC_EXACT this does not reproduce the canonical fp32
// order of DESIGN.md R1: a code bit may differ from the oracle's where |y_j| <= 1e-5 ||x||, f_scale within 1e-5
// relative (guard band of SURVEY.md 8(c) C1, checked in tests/test_gpu_parity.py::test_encode_fast_guard_band).
//
// One CTA = 8 warps x 16 tokens.  P_hi / P_lo live in shared memory as row-major bf16 [i][j] (XOR-swizzled 16-byte
// chunks) and are read as B fragments with ldmatrix.trans; the CTA stages them once and then loops over its token
// tiles (grid.x CTAs per (sequence, KV head)), so P is read from L2 a few hundred times, not once per tile.  The raw K
// tile is staged with cp.async; the A fragments (x_hi, x_lo) are built per k-step in registers.
#include "rbq_common.cuh"

namespace {

constexpr int EF_WARPS = 8;
constexpr int EF_THREADS = EF_WARPS * 32;
constexpr int EF_TOK = EF_WARPS * 16;                       // tokens per tile
constexpr int EF_KPITCH = RBQ_D * 2 + 16;                   // bytes per staged bf16 K row (+16: conflict-free fragment reads)
constexpr int EF_SMEM = 2 * RBQ_D * RBQ_D * 2 + EF_TOK * EF_KPITCH + RBQ_D * 4;   // P_hi, P_lo, K tile, c_k

__device__ __forceinline__ uint32_t ef_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ef_ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ef_mma(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// (v0, v1) -> packed bf16 hi parts and packed bf16 lo parts (lo = bf16(v - hi))
__device__ __forceinline__ void ef_split(float v0, float v1, uint32_t& hi, uint32_t& lo) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  const __nv_bfloat162 l = __floats2bfloat162_rn(v0 - rbq_bf16lo(hi), v1 - rbq_bf16hi(hi));
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// grid = (tiles-per-group CTAs, B*Hkv).  Tokens [t_begin[b], t_begin[b] + count[b]) of every (b, kv head).
__global__ void __launch_bounds__(EF_THREADS, 2)
encode_fast_kernel(const __nv_bfloat16* __restrict__ K, long long sb, long long sh, long long st,
                   const int32_t* __restrict__ t_begin, const int32_t* __restrict__ t_count, int fixed_count, int Hkv,
                   int Lcap, const float* __restrict__ rot, const float* __restrict__ c_k, uint32_t* __restrict__ codes,
                   float* __restrict__ f_scale) {
  extern __shared__ __align__(128) unsigned char ef_smem[];
  unsigned char* s_ph = ef_smem;                              // P_hi bf16 [128][128], 16-byte chunk c of row i at (c ^ (i & 7))
  unsigned char* s_pl = ef_smem + RBQ_D * RBQ_D * 2;
  unsigned char* s_k = ef_smem + 2 * RBQ_D * RBQ_D * 2;       // raw K tile [EF_TOK][EF_KPITCH]
  float* s_ck = reinterpret_cast<float*>(s_k + EF_TOK * EF_KPITCH);

  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int tb = t_begin ? t_begin[b] : 0;
  const int cnt = t_count ? t_count[b] : fixed_count;
  if ((int)blockIdx.x * EF_TOK >= cnt) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g4 = lane >> 2, t4 = lane & 3;

  // P -> bf16 hi / lo, row-major, swizzled (once per CTA)
  for (int e = tid; e < RBQ_D * RBQ_D / 2; e += EF_THREADS) {
    const int i = e >> 6, j2 = (e & 63) * 2;                  // two consecutive outputs j2, j2 + 1 of input row i
    const float2 v = __ldg(reinterpret_cast<const float2*>(rot + i * RBQ_D + j2));
    uint32_t hi, lo;
    ef_split(v.x, v.y, hi, lo);
    const int off = i * 256 + ((((j2 >> 3) ^ (i & 7)) << 4) | ((j2 & 7) * 2));
    *reinterpret_cast<uint32_t*>(s_ph + off) = hi;
    *reinterpret_cast<uint32_t*>(s_pl + off) = lo;
  }
  if (tid < RBQ_D) s_ck[tid] = c_k[(size_t)bg * RBQ_D + tid];

  const __nv_bfloat16* base = K + (long long)b * sb + (long long)g * sh + (long long)tb * st;
  const uint32_t ph = ef_smem_u32(s_ph), pl = ef_smem_u32(s_pl), sk = ef_smem_u32(s_k);

  for (int tile0 = (int)blockIdx.x * EF_TOK; tile0 < cnt; tile0 += (int)gridDim.x * EF_TOK) {
    const int ntok = min(EF_TOK, cnt - tile0);
    __syncthreads();                                          // previous tile consumed (and P / c_k staged on the first pass)
    for (int e = tid; e < EF_TOK * 16; e += EF_THREADS) {     // raw K rows, 16-byte pieces
      const int r = e >> 4, c = e & 15;
      if (r < ntok)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sk + (uint32_t)(r * EF_KPITCH + c * 16)),
                     "l"(base + (long long)(tile0 + r) * st + c * 8) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();

    const int r0 = warp * 16 + g4, r1 = r0 + 8;               // this lane's two token rows inside the tile
    const bool ok0 = r0 < ntok, ok1 = r1 < ntok;
    float acc[16][4];
#pragma unroll
    for (int nt = 0; nt < 16; ++nt) { acc[nt][0] = 0.f; acc[nt][1] = 0.f; acc[nt][2] = 0.f; acc[nt][3] = 0.f; }
    float n2a = 0.0f, n2b = 0.0f;
#pragma unroll 1
    for (int ks = 0; ks < 8; ++ks) {
      // A fragments of k-step ks: x = k - c_k at columns 16 ks + 2 t4 (+1) and + 8 (+9), rows r0 / r1
      uint32_t ah[4], al[4];
      const int c0 = 16 * ks + 2 * t4;
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        const int col = c0 + 8 * half;
        const float ck0 = s_ck[col], ck1 = s_ck[col + 1];
        const uint32_t ka = ok0 ? *reinterpret_cast<const uint32_t*>(s_k + r0 * EF_KPITCH + col * 2) : 0u;
        const uint32_t kb = ok1 ? *reinterpret_cast<const uint32_t*>(s_k + r1 * EF_KPITCH + col * 2) : 0u;
        const float xa0 = ok0 ? rbq_bf16lo(ka) - ck0 : 0.f, xa1 = ok0 ? rbq_bf16hi(ka) - ck1 : 0.f;
        const float xb0 = ok1 ? rbq_bf16lo(kb) - ck0 : 0.f, xb1 = ok1 ? rbq_bf16hi(kb) - ck1 : 0.f;
        n2a = fmaf(xa0, xa0, n2a); n2a = fmaf(xa1, xa1, n2a);
        n2b = fmaf(xb0, xb0, n2b); n2b = fmaf(xb1, xb1, n2b);
        ef_split(xa0, xa1, ah[2 * half], al[2 * half]);
        ef_split(xb0, xb1, ah[2 * half + 1], al[2 * half + 1]);
      }
      // B fragments: P rows 16 ks .. 16 ks + 15 (k), 16 output columns per ldmatrix.x4.trans
#pragma unroll
      for (int c2 = 0; c2 < 8; ++c2) {
        const int row = 16 * ks + (lane & 7) + ((lane >> 3) & 1) * 8, ch = 2 * c2 + (lane >> 4);
        const uint32_t off = (uint32_t)(row * 256 + ((ch ^ (row & 7)) << 4));
        uint32_t bh[4], bl[4];
        ef_ldsm_x4_t(bh, ph + off);
        ef_ldsm_x4_t(bl, pl + off);
        ef_mma(acc[2 * c2], ah, bh[0], bh[1]);
        ef_mma(acc[2 * c2 + 1], ah, bh[2], bh[3]);
        ef_mma(acc[2 * c2], al, bh[0], bh[1]);
        ef_mma(acc[2 * c2 + 1], al, bh[2], bh[3]);
        ef_mma(acc[2 * c2], ah, bl[0], bl[1]);
        ef_mma(acc[2 * c2 + 1], ah, bl[2], bl[3]);
      }
    }
    // epilogue: l1, sign bits (bit j % 32 of word j / 32 = [y_j > 0]), f_scale = ||x||^2 / ||y||_1
    float l1a = 0.0f, l1b = 0.0f;
    uint32_t wa[RBQ_WORDS] = {0u, 0u, 0u, 0u}, wb[RBQ_WORDS] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int nt = 0; nt < 16; ++nt) {
      const int sh2 = 8 * (nt & 3) + 2 * t4;
      l1a += fabsf(acc[nt][0]) + fabsf(acc[nt][1]);
      l1b += fabsf(acc[nt][2]) + fabsf(acc[nt][3]);
      wa[nt >> 2] |= ((acc[nt][0] > 0.f ? 1u : 0u) << sh2) | ((acc[nt][1] > 0.f ? 1u : 0u) << (sh2 + 1));
      wb[nt >> 2] |= ((acc[nt][2] > 0.f ? 1u : 0u) << sh2) | ((acc[nt][3] > 0.f ? 1u : 0u) << (sh2 + 1));
    }
#pragma unroll
    for (int o = 1; o < 4; o <<= 1) {
      l1a += __shfl_xor_sync(0xffffffffu, l1a, o); l1b += __shfl_xor_sync(0xffffffffu, l1b, o);
      n2a += __shfl_xor_sync(0xffffffffu, n2a, o); n2b += __shfl_xor_sync(0xffffffffu, n2b, o);
#pragma unroll
      for (int w = 0; w < RBQ_WORDS; ++w) {
        wa[w] |= __shfl_xor_sync(0xffffffffu, wa[w], o);
        wb[w] |= __shfl_xor_sync(0xffffffffu, wb[w], o);
      }
    }
    if (t4 == 0) {
      const size_t tok = (size_t)bg * Lcap + tb + tile0;
      if (ok0) {
        reinterpret_cast<uint4*>(codes)[tok + r0] = make_uint4(wa[0], wa[1], wa[2], wa[3]);
        f_scale[tok + r0] = (l1a == 0.0f) ? 0.0f : n2a / l1a;
      }
      if (ok1) {
        reinterpret_cast<uint4*>(codes)[tok + r1] = make_uint4(wb[0], wb[1], wb[2], wb[3]);
        f_scale[tok + r1] = (l1b == 0.0f) ? 0.0f : n2b / l1b;
      }
    }
  }
}

}  // namespace

int rbq_launch_encode_fast(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count, int fixed_count,
                           int max_count, const rbq_index* idx, cudaStream_t s) {
  static bool attr_set = false;
  if (!attr_set) {
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(encode_fast_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, EF_SMEM));
    attr_set = true;
  }
  const int BG = ctx->cfg.batch * ctx->cfg.n_kv_heads;
  const int tiles = (max_count + EF_TOK - 1) / EF_TOK;
  int gx = (2 * ctx->sm_count + BG - 1) / BG;                 // about two CTAs per SM in total; each loops over its tiles
  gx = gx < 1 ? 1 : (gx > tiles ? tiles : gx);
  encode_fast_kernel<<<dim3(gx, BG), EF_THREADS, EF_SMEM, s>>>((const __nv_bfloat16*)kv.k, kv.sb, kv.sh, kv.st, t_begin, t_count,
                                                              fixed_count, ctx->cfg.n_kv_heads, ctx->cfg.max_tokens,
                                                              ctx->cfg.rot, idx->c_k, idx->codes, idx->f_scale);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
