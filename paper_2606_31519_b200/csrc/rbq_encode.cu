// rbq_encode.cu -- S1/S2: centroid, Alg.1 index construction (PAPER.md:L106-147, L149-151,
// L485-487), cache-tail append (L215).
//
// RBQ_ENC_EXACT reproduces the canonical fp32 order of DESIGN.md R1 bit for bit:
//   x_i = fl32(k_i) - c_k,i ; n2 <- fmaf(x_i, x_i, n2), i ascending ;
//   dense: y_j <- fmaf(x_i, P[i][j], y_j), i ascending, one accumulator per j
//          (a non-split-K SGEMM inner loop, here register-tiled 4 tokens x 8 outputs per thread);
//   WH   : u = s.*x ; butterflies h = 1,2,..,D/2, (a,b) -> (a+b, a-b) ; y = u * fl32(1/sqrt(D)) ;
//   l1 <- l1 + |y_j| (WH: |u_j|, then * fl32(1/sqrt(D))), j ascending ; f_scale = n2 / l1 (IEEE).
// The file is compiled with -fmad=false; every fused multiply-add below is an explicit fmaf().
#include "rbq_common.cuh"

namespace {

constexpr int ENC_TOK = 64;        // tokens per CTA tile
constexpr int ENC_THREADS = 256;
// head_dim D is a template parameter (64, 128, 256).  XS = D + 1: padded row stride of the x / y tile (bank-conflict-free
// per-token access).  The dense P is staged in chunks of KC = min(D, 128) rows (D = 256: two chunks of 128 KB).

// ---- centroid: c_k = mean over t < n of K[b][g][t][:] , fp64 accumulation ------------------------
// Partial sums over CEN_SPLIT contiguous token ranges, then a fixed-order final sum.  fp64 sums of
// bf16 / fp32 inputs of this size are exact (or within 1 ulp of fp64), so the fp32 result is the
// correctly rounded mean irrespective of the order.
constexpr int CEN_SPLIT = 64;

// 8 consecutive elements of a row as floats (16-byte loads for bf16, 2 x 16 bytes for fp32)
__device__ __forceinline__ void rbq_ld8(const __nv_bfloat16* p, float (&v)[8]) {
  const uint4 u = __ldg(reinterpret_cast<const uint4*>(p));
  v[0] = rbq_bf16lo(u.x); v[1] = rbq_bf16hi(u.x); v[2] = rbq_bf16lo(u.y); v[3] = rbq_bf16hi(u.y);
  v[4] = rbq_bf16lo(u.z); v[5] = rbq_bf16hi(u.z); v[6] = rbq_bf16lo(u.w); v[7] = rbq_bf16hi(u.w);
}
__device__ __forceinline__ void rbq_ld8(const float* p, float (&v)[8]) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(p)), b = __ldg(reinterpret_cast<const float4*>(p) + 1);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}

// raw 8-element pieces (kept unconverted while in flight: 4 registers for bf16, 8 for fp32)
struct RbqRaw8F { float4 a, b; };
__device__ __forceinline__ uint4 rbq_ldraw8(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
__device__ __forceinline__ RbqRaw8F rbq_ldraw8(const float* p) {
  return {__ldg(reinterpret_cast<const float4*>(p)), __ldg(reinterpret_cast<const float4*>(p) + 1)};
}
__device__ __forceinline__ uint4 rbq_zero_raw(const __nv_bfloat16*) { return make_uint4(0u, 0u, 0u, 0u); }
__device__ __forceinline__ RbqRaw8F rbq_zero_raw(const float*) { return {make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)}; }
__device__ __forceinline__ void rbq_raw_to_f(const uint4& u, float (&v)[8]) {
  v[0] = rbq_bf16lo(u.x); v[1] = rbq_bf16hi(u.x); v[2] = rbq_bf16lo(u.y); v[3] = rbq_bf16hi(u.y);
  v[4] = rbq_bf16lo(u.z); v[5] = rbq_bf16hi(u.z); v[6] = rbq_bf16lo(u.w); v[7] = rbq_bf16hi(u.w);
}
__device__ __forceinline__ void rbq_raw_to_f(const RbqRaw8F& u, float (&v)[8]) {
  v[0] = u.a.x; v[1] = u.a.y; v[2] = u.a.z; v[3] = u.a.w; v[4] = u.b.x; v[5] = u.b.y; v[6] = u.b.z; v[7] = u.b.w;
}

// grid = (B*Hkv, CEN_SPLIT), 256 threads: 16 threads per row (8 dims each), 16 rows per round, CEN_FLIGHT rounds (raw
// 16-byte pieces) in flight per thread; 4 CTAs per SM keep ~19 MB in flight over the chip.
constexpr int CEN_THREADS = 256;

template <typename T, int D>
__global__ void __launch_bounds__(CEN_THREADS, D == 256 ? 2 : 4)
centroid_partial_kernel(const T* __restrict__ K, long long sb, long long sh, long long st,
                        const int32_t* __restrict__ seq_lens, int Hkv, double* __restrict__ part) {
  constexpr int TPR = D / 8, RPR = CEN_THREADS / TPR;          // threads per row (8 dims each), rows per round
  __shared__ double s_acc[RPR][D];
  const int bg = blockIdx.x, b = bg / Hkv, g = bg % Hkv, s = blockIdx.y;
  const int c8 = (threadIdx.x % TPR) * 8, r = threadIdx.x / TPR;
  const int n = seq_lens[b];
  const int per = (n + CEN_SPLIT - 1) / CEN_SPLIT;
  const int t0 = s * per, t1 = min(n, t0 + per);
  const T* base = K + (long long)b * sb + (long long)g * sh + c8;
  constexpr int CEN_FLIGHT = sizeof(T) == 2 ? 8 : 2;          // 32 / 16 registers of raw data in flight
  double acc[8];
#pragma unroll
  for (int d = 0; d < 8; ++d) acc[d] = 0.0;
  for (int t = t0 + r; t < t1; t += CEN_FLIGHT * RPR) {
    decltype(rbq_ldraw8(base)) raw[CEN_FLIGHT];
#pragma unroll
    for (int u = 0; u < CEN_FLIGHT; ++u) {
      const int tt = t + u * RPR;
      raw[u] = (tt < t1) ? rbq_ldraw8(base + (long long)tt * st) : rbq_zero_raw(base);
    }
#pragma unroll
    for (int u = 0; u < CEN_FLIGHT; ++u) {
      float v[8];
      rbq_raw_to_f(raw[u], v);
#pragma unroll
      for (int d = 0; d < 8; ++d) acc[d] += (double)v[d];
    }
  }
#pragma unroll
  for (int d = 0; d < 8; ++d) s_acc[r][c8 + d] = acc[d];
  __syncthreads();
  if (threadIdx.x < D) {
    double a = 0.0;
#pragma unroll
    for (int k = 0; k < RPR; ++k) a += s_acc[k][threadIdx.x];
    part[((size_t)bg * CEN_SPLIT + s) * D + threadIdx.x] = a;
  }
}

__global__ void centroid_final_kernel(const double* __restrict__ part, const int32_t* __restrict__ seq_lens,
                                      int Hkv, int D, float* __restrict__ c_k) {      // D threads
  const int bg = blockIdx.x, b = bg / Hkv, d = threadIdx.x;
  const int n = seq_lens[b];
  double acc = 0.0;
  for (int s = 0; s < CEN_SPLIT; ++s) acc += part[((size_t)bg * CEN_SPLIT + s) * D + d];
  c_k[(size_t)bg * D + d] = (n > 0) ? (float)(acc / (double)n) : 0.0f;
}

// ---- Alg.1 tile kernel --------------------------------------------------------------------------
// grid = (ceil(max_count / ENC_TOK), B*Hkv).  Tokens [t_begin[b], t_begin[b]+count[b]).
// smem: x tile [ENC_TOK][XS] fp32 (becomes the y tile), n2[ENC_TOK], P chunk [KC][D] fp32 (dense) or the D signs (WH).
template <typename T, int ROT, int D>
__global__ void __launch_bounds__(ENC_THREADS)
encode_kernel(const T* __restrict__ K, long long sb, long long sh, long long st,
              const int32_t* __restrict__ t_begin, const int32_t* __restrict__ t_count, int fixed_count,
              int Hkv, int Lcap, const float* __restrict__ rot, const float* __restrict__ c_k,
              uint32_t* __restrict__ codes, void* __restrict__ f_scale, int fs_f16) {
  constexpr int XS = D + 1, W = D / 32, KC = D < 128 ? D : 128, NG = D / 64;   // NG: float4 output groups per thread
  extern __shared__ __align__(16) float smem[];
  float* xs = smem;                                 // [ENC_TOK][XS]
  float* n2s = xs + ENC_TOK * XS;                   // [ENC_TOK]
  float* rs = n2s + ENC_TOK;                        // dense: [KC][D]; WH: [D] signs

  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int tb = t_begin ? t_begin[b] : 0;
  const int cnt = min(t_count ? t_count[b] : fixed_count, Lcap - tb);   // never past the capacity (append overflow, rbq_status_flags)
  const int tile0 = blockIdx.x * ENC_TOK;
  if (tile0 >= cnt) return;
  const int ntok = min(ENC_TOK, cnt - tile0);
  const int tid = threadIdx.x;
  const T* base = K + (long long)b * sb + (long long)g * sh + (long long)(tb + tile0) * st;
  const float* ck = c_k + (size_t)bg * D;

  // x = fl32(k) - c_k
  // 16-byte loads; a warp covers 8 rows x 4 chunks of 8 elements so that its shared-memory stores are conflict-free
  // with the padded row stride (bank = row + 8 * chunk + k)
  for (int e = tid; e < ENC_TOK * D / 8; e += ENC_THREADS) {
    const int wv = e >> 5, ln = e & 31;
    const int r = (wv / (D / 32)) * 8 + (ln >> 2), d = ((wv % (D / 32)) * 4 + (ln & 3)) * 8;
    float v[8];
    if (r < ntok) rbq_ld8(base + (long long)r * st + d, v);
#pragma unroll
    for (int k = 0; k < 8; ++k) xs[r * XS + d + k] = (r < ntok) ? __fsub_rn(v[k], ck[d + k]) : 0.0f;
  }
  if (ROT == RBQ_ROT_WH && tid < D) rs[tid] = rot[tid];
  __syncthreads();

  // n2: one thread per token, sequential fma chain (i ascending)
  if (tid < ENC_TOK) {
    float n2 = 0.0f;
    const float* xr = xs + tid * XS;
#pragma unroll 8
    for (int i = 0; i < D; ++i) n2 = fmaf(xr[i], xr[i], n2);
    n2s[tid] = n2;
  }

  if (ROT == RBQ_ROT_DENSE) {
    // thread -> 4 tokens (tt*4..+3) x 4*NG outputs (columns 64 q + tj*4 .. +3, q < NG); P staged KC rows at a time, the
    // chains run on across the chunks (i ascending: the canonical order)
    const int tj = tid & 15, tt = tid >> 4;
    float acc[4][4 * NG];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = 0; n < 4 * NG; ++n) acc[m][n] = 0.0f;
    const float* x0 = xs + (tt * 4) * XS;
    for (int ic = 0; ic < D; ic += KC) {
      if (ic > 0) __syncthreads();                  // everyone done with the previous chunk of P
      for (int e = tid; e < KC * D / 4; e += ENC_THREADS)
        reinterpret_cast<float4*>(rs)[e] = reinterpret_cast<const float4*>(rot + (size_t)ic * D)[e];
      __syncthreads();
#pragma unroll 4
      for (int i = 0; i < KC; ++i) {
        float rr[4 * NG];
#pragma unroll
        for (int q = 0; q < NG; ++q) {
          const float4 r4 = *reinterpret_cast<const float4*>(rs + i * D + 64 * q + tj * 4);
          rr[4 * q] = r4.x; rr[4 * q + 1] = r4.y; rr[4 * q + 2] = r4.z; rr[4 * q + 3] = r4.w;
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const float xv = x0[m * XS + ic + i];
#pragma unroll
          for (int n = 0; n < 4 * NG; ++n) acc[m][n] = fmaf(xv, rr[n], acc[m][n]);
        }
      }
    }
    __syncthreads();                                 // everyone done reading x (n2 included)
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = 0; n < 4 * NG; ++n)
        xs[(tt * 4 + m) * XS + 64 * (n >> 2) + tj * 4 + (n & 3)] = acc[m][n];
  } else {
    __syncthreads();
    // WH: warp w handles tokens w, w+8, ...; lane holds elements W*lane .. W*lane + W-1: levels h < W inside the lane, the
    // others by shuffles
    const int warp = tid >> 5, lane = tid & 31;
    for (int r = warp; r < ENC_TOK; r += ENC_THREADS / 32) {
      float* xr = xs + r * XS + lane * W;
      float u[W];
#pragma unroll
      for (int e = 0; e < W; ++e) u[e] = __fmul_rn(rs[lane * W + e], xr[e]);
#pragma unroll
      for (int hh = 1; hh < W; hh <<= 1) {
#pragma unroll
        for (int e = 0; e < W; ++e) {
          if ((e & hh) == 0) {
            const float a = u[e], c = u[e | hh];
            u[e] = __fadd_rn(a, c);
            u[e | hh] = __fsub_rn(a, c);
          }
        }
      }
#pragma unroll
      for (int m = 1; m < 32; m <<= 1) {                                      // h = W*m
        // (a, b) -> (a + b, a - b): the upper lane computes p - u, the lower one u + p; both are fmaf(u, +-1, p),
        // bit-identical to the add / subtract (the product with +-1 is exact, one rounding)
        const float sg = (lane & m) ? -1.0f : 1.0f;
#pragma unroll
        for (int e = 0; e < W; ++e) {
          const float pp = __shfl_xor_sync(0xffffffffu, u[e], m);
          u[e] = fmaf(u[e], sg, pp);
        }
      }
      __syncwarp();
#pragma unroll
      for (int e = 0; e < W; ++e) xr[e] = u[e];                              // unscaled u
    }
  }
  __syncthreads();

  // epilogue: one thread per token: l1 (sequential), sign bits, f_scale
  if (tid < ntok) {
    const float* yr = xs + tid * XS;
    float l1 = 0.0f;
    uint32_t w[W];
    const float c = (float)(1.0 / sqrt((double)D));
#pragma unroll
    for (int ww = 0; ww < W; ++ww) {
      uint32_t word = 0;
#pragma unroll 8
      for (int j = 0; j < 32; ++j) {
        const float yv = yr[ww * 32 + j];
        l1 = __fadd_rn(l1, fabsf(yv));
        const float ys = (ROT == RBQ_ROT_DENSE) ? yv : __fmul_rn(yv, c);
        word |= (ys > 0.0f ? 1u : 0u) << j;
      }
      w[ww] = word;
    }
    if (ROT == RBQ_ROT_WH) l1 = __fmul_rn(l1, c);
    const size_t tok = (size_t)bg * Lcap + tb + tile0 + tid;
    if (W == 2) {
      reinterpret_cast<uint2*>(codes)[tok] = make_uint2(w[0], w[1]);
    } else {
#pragma unroll
      for (int q = 0; q < W / 4; ++q)
        reinterpret_cast<uint4*>(codes)[tok * (W / 4) + q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
    }
    rbq_store_factor(f_scale, fs_f16, tok, (l1 == 0.0f) ? 0.0f : __fdiv_rn(n2s[tid], l1));
  }
}

// f_bias[b][hq][t] = <c_q[b][hq], k_t> ("<c_q,k> ... can all be pre-calculated"), one canonical fma chain
// per (token, query head), i ascending (R1) -- bit-identical to the oracle in both encode modes.
// grid = (ceil(max_count / FB_TOK), B*Hkv), FB_TOK threads: the K rows of FB_TOK tokens are staged in shared memory with
// coalesced 16-byte loads (padded rows: conflict-free per-token reads), c_q of the group's G heads next to them; a
// thread owns one token and runs the G chains side by side (each staged k_i feeds G independent FMAs).
constexpr int FB_TOK = 128;

template <typename T, int D>
__global__ void __launch_bounds__(FB_TOK)
fbias_kernel(const T* __restrict__ K, long long sb, long long sh, long long st, const int32_t* __restrict__ t_begin,
             const int32_t* __restrict__ t_count, int fixed_count, int Hq, int Hkv, int Lcap, const float* __restrict__ c_q,
             float* __restrict__ f_bias) {
  constexpr int FB_XS = D + 1;
  extern __shared__ __align__(16) float fb_smem[];
  float* ks = fb_smem;                              // [FB_TOK][FB_XS]
  float* cq = ks + FB_TOK * FB_XS;                  // [G][D]
  const int G = Hq / Hkv;
  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int tb = t_begin ? t_begin[b] : 0;
  const int cnt = min(t_count ? t_count[b] : fixed_count, Lcap - tb);
  const int tile0 = blockIdx.x * FB_TOK;
  if (tile0 >= cnt) return;
  const int ntok = min(FB_TOK, cnt - tile0);
  const int tid = threadIdx.x;
  const T* base = K + (long long)b * sb + (long long)g * sh + (long long)(tb + tile0) * st;
  for (int e = tid; e < FB_TOK * D / 8; e += FB_TOK) {
    const int wv = e >> 5, ln = e & 31;
    const int r = (wv / (D / 32)) * 8 + (ln >> 2), d = ((wv % (D / 32)) * 4 + (ln & 3)) * 8;
    float v[8];
    if (r < ntok) rbq_ld8(base + (long long)r * st + d, v);
#pragma unroll
    for (int k = 0; k < 8; ++k) ks[r * FB_XS + d + k] = (r < ntok) ? v[k] : 0.0f;
  }
  for (int e = tid; e < G * D; e += FB_TOK) cq[e] = c_q[((size_t)b * Hq + (size_t)g * G) * D + e];
  __syncthreads();
  if (tid >= ntok) return;
  const float* kr = ks + tid * FB_XS;
  float acc[RBQ_MAX_G];
#pragma unroll
  for (int h = 0; h < RBQ_MAX_G; ++h) acc[h] = 0.0f;
#pragma unroll 8
  for (int i = 0; i < D; ++i) {
    const float kv = kr[i];
#pragma unroll
    for (int h = 0; h < RBQ_MAX_G; ++h)
      if (h < G) acc[h] = fmaf(cq[h * D + i], kv, acc[h]);
  }
#pragma unroll
  for (int h = 0; h < RBQ_MAX_G; ++h)
    if (h < G) f_bias[((size_t)b * Hq + (size_t)g * G + h) * Lcap + tb + tile0 + tid] = acc[h];
}

__global__ void set_counts_kernel(const int32_t* __restrict__ seq_lens, int32_t* n_indexed, int32_t* n_total, int B) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < B) { n_indexed[b] = seq_lens[b]; n_total[b] = seq_lens[b]; }
}

// S2: commit an earlier flush (n_indexed += commit), copy n_new rows per (b, kv head) to the cache tail
// [n_total, n_total + n_new), then n_total += n_new (append_bump_kernel, launched after the copy).  16-byte vector copies.
// Rows that would land at or beyond the capacity Lcap are dropped and the sticky RBQ_FLAG_APPEND_OVERFLOW bit is set
// (rbq_status_flags): the counts never exceed Lcap, so no later stage indexes past an allocation.
__global__ void append_copy_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new, int n_new,
                                   int row_vec, char* __restrict__ kc, char* __restrict__ vc, long long sb_bytes,
                                   long long sh_bytes, long long st_bytes, int Hkv, int Lcap,
                                   const int32_t* __restrict__ n_total) {
  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n_new * row_vec) return;
  const int r = e / row_vec, c = e % row_vec;
  const int t = n_total[b] + r;
  if (t >= Lcap) return;
  const long long dst = (long long)b * sb_bytes + (long long)g * sh_bytes + (long long)t * st_bytes + c * 16;
  const size_t src = ((size_t)bg * n_new + r) * row_vec + c;
  *reinterpret_cast<uint4*>(kc + dst) = k_new[src];
  *reinterpret_cast<uint4*>(vc + dst) = v_new[src];
}

__global__ void append_bump_kernel(int32_t* n_indexed, int32_t* n_total, int B, int commit, int n_new, int Lcap,
                                   uint32_t* __restrict__ flags) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < B) {
    int nt = n_total[b] + n_new;
    if (nt > Lcap) { nt = Lcap; atomicOr(flags, RBQ_FLAG_APPEND_OVERFLOW); }
    n_total[b] = nt;
    n_indexed[b] = min(n_indexed[b] + commit, nt);
  }
}

}  // namespace

template <typename T, int D>
static int launch_centroid_t(rbq_ctx* ctx, const RbqKV& kv, const int32_t* seq_lens, float* c_k, cudaStream_t s) {
  const int BG = ctx->cfg.batch * ctx->cfg.n_kv_heads;
  double* part = reinterpret_cast<double*>(static_cast<char*>(ctx->ws) + ctx->off_centroid);
  centroid_partial_kernel<T, D><<<dim3(BG, CEN_SPLIT), CEN_THREADS, 0, s>>>((const T*)kv.k, kv.sb, kv.sh, kv.st, seq_lens,
                                                                           ctx->cfg.n_kv_heads, part);
  RBQ_LAUNCH_OK(ctx);
  centroid_final_kernel<<<BG, D, 0, s>>>(part, seq_lens, ctx->cfg.n_kv_heads, D, c_k);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

// dispatch on (K/V dtype, head_dim): F<T, D>(args...)
#define RBQ_DISPATCH_TD(ctx, F, ...)                                                              \
  do {                                                                                            \
    const bool bf_ = (ctx)->cfg.kv_dtype == RBQ_BF16;                                             \
    switch ((ctx)->cfg.head_dim) {                                                                \
      case 64: return bf_ ? F<__nv_bfloat16, 64>(__VA_ARGS__) : F<float, 64>(__VA_ARGS__);         \
      case 256: return bf_ ? F<__nv_bfloat16, 256>(__VA_ARGS__) : F<float, 256>(__VA_ARGS__);      \
      default: return bf_ ? F<__nv_bfloat16, 128>(__VA_ARGS__) : F<float, 128>(__VA_ARGS__);       \
    }                                                                                             \
  } while (0)

int rbq_launch_centroid(rbq_ctx* ctx, const RbqKV& kv, const int32_t* seq_lens, float* c_k, cudaStream_t s) {
  RBQ_DISPATCH_TD(ctx, launch_centroid_t, ctx, kv, seq_lens, c_k, s);
}

template <typename T, int D, int ROT>
static int launch_encode_r(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count,
                           int fixed_count, int max_count, const rbq_index* idx, cudaStream_t s) {
  constexpr int KC = D < 128 ? D : 128;
  const size_t smem = (size_t)(ENC_TOK * (D + 1) + ENC_TOK + (ROT == RBQ_ROT_DENSE ? KC * D : D)) * sizeof(float);
  auto kern = encode_kernel<T, ROT, D>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_ENC_EXACT + (D == 64 ? 0 : D == 128 ? 4 : 8) + (sizeof(T) == 2 ? 0 : 2) + (ROT == RBQ_ROT_DENSE ? 0 : 1), kern, smem);
  dim3 grid((max_count + ENC_TOK - 1) / ENC_TOK, ctx->cfg.batch * ctx->cfg.n_kv_heads);
  kern<<<grid, ENC_THREADS, smem, s>>>((const T*)kv.k, kv.sb, kv.sh, kv.st, t_begin, t_count, fixed_count,
                                       ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, ctx->cfg.rot, idx->c_k,
                                       idx->codes, idx->f_scale, ctx->cfg.factor_dtype == RBQ_F16 ? 1 : 0);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

template <typename T, int D>
static int launch_encode_t(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count,
                           int fixed_count, int max_count, const rbq_index* idx, cudaStream_t s) {
  if (ctx->cfg.rot_kind == RBQ_ROT_WH) return launch_encode_r<T, D, RBQ_ROT_WH>(ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
  return launch_encode_r<T, D, RBQ_ROT_DENSE>(ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
}

// f_bias = <c_q, k> for the same token ranges (either encode mode)
template <typename T, int D>
static int launch_fbias_t(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count, int fixed_count,
                          int max_count, const rbq_index* idx, cudaStream_t s) {
  const size_t smem = (size_t)(FB_TOK * (D + 1) + ctx->G * D) * sizeof(float);
  auto kern = fbias_kernel<T, D>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_FBIAS + (D == 64 ? 0 : D == 128 ? 2 : 4) + (sizeof(T) == 2 ? 0 : 1), kern, smem);
  dim3 grid((max_count + FB_TOK - 1) / FB_TOK, ctx->cfg.batch * ctx->cfg.n_kv_heads);
  kern<<<grid, FB_TOK, smem, s>>>((const T*)kv.k, kv.sb, kv.sh, kv.st, t_begin, t_count, fixed_count, ctx->cfg.n_q_heads,
                                  ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, idx->c_q, idx->f_bias);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

static int launch_encode_exact(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count, int fixed_count,
                               int max_count, const rbq_index* idx, cudaStream_t s) {
  RBQ_DISPATCH_TD(ctx, launch_encode_t, ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
}
static int launch_fbias(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count, int fixed_count,
                        int max_count, const rbq_index* idx, cudaStream_t s) {
  RBQ_DISPATCH_TD(ctx, launch_fbias_t, ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
}

int rbq_launch_encode(rbq_ctx* ctx, const RbqKV& kv, const int32_t* t_begin, const int32_t* t_count,
                      int fixed_count, int max_count, const rbq_index* idx, cudaStream_t s) {
  if (max_count <= 0) return RBQ_OK;
  const int rc = ctx->cfg.enc_mode == RBQ_ENC_FAST ? rbq_launch_encode_fast(ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s)
                                                   : launch_encode_exact(ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
  if (rc != RBQ_OK || !idx->c_q) return rc;
  return launch_fbias(ctx, kv, t_begin, t_count, fixed_count, max_count, idx, s);
}

int rbq_launch_set_counts(rbq_ctx* ctx, const int32_t* seq_lens, int32_t* n_indexed, int32_t* n_total, cudaStream_t s) {
  set_counts_kernel<<<(ctx->cfg.batch + 127) / 128, 128, 0, s>>>(seq_lens, n_indexed, n_total, ctx->cfg.batch);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

int rbq_launch_append_copy(rbq_ctx* ctx, const void* k_new, const void* v_new, int n_new, const RbqKV& kv,
                           int32_t* n_indexed, int32_t* n_total, int commit, cudaStream_t s) {
  const int esz = ctx->cfg.kv_dtype == RBQ_BF16 ? 2 : 4;
  const int row_vec = ctx->cfg.head_dim * esz / 16;
  if (n_new > 0) {
    dim3 grid((n_new * row_vec + 127) / 128, ctx->cfg.batch * ctx->cfg.n_kv_heads);
    append_copy_kernel<<<grid, 128, 0, s>>>((const uint4*)k_new, (const uint4*)v_new, n_new, row_vec,
                                            (char*)kv.k, (char*)kv.v, kv.sb * esz, kv.sh * esz, kv.st * esz,
                                            ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, n_total);
    RBQ_LAUNCH_OK(ctx);
  }
  append_bump_kernel<<<(ctx->cfg.batch + 127) / 128, 128, 0, s>>>(n_indexed, n_total, ctx->cfg.batch, commit, n_new, ctx->cfg.max_tokens,
                                                                  reinterpret_cast<uint32_t*>(static_cast<char*>(ctx->ws) + ctx->off_flags));
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
