// rbq_attention.cu -- S7: exact attention over the gathered selected tokens and the pending window
// (Alg.2 lines 14-15, L188-190; L215 "K_local ... participate in the hybrid attention";
// renormalised over the attended set, R7).
//
// HBM-bound gather of 2*D*sizeof(T) bytes per attended (token, q head) with ~4*D FLOP per row:
// far below any compute roof, so the contraction stays on the FP32 pipe (no tensor cores) and the
// design is about bytes in flight: flash-decoding split-K over the per-row index list, work = fixed
// 256-token chunks of (sel_idx[row] ++ pending), distributed over a persistent grid sized from the
// SM count; each half-warp reads one 256-byte K (then V) row per 128-bit load instruction, 8 rows
// per warp in flight per operand; (m, l, o) partials per chunk, then a per-row merge.
#include "rbq_common.cuh"

namespace {

constexpr int AT_THREADS = 256;
constexpr int AT_WARPS = AT_THREADS / 32;
constexpr int AT_CHUNK = AT_WARPS * 32;       // tokens per chunk: one 32-token strip per warp
constexpr int AT_PART = RBQ_D + 2;            // floats per partial: o[128], m, l
constexpr int AT_MAX_ROWS = 4096;

struct Row8 { float v[8]; };

__device__ __forceinline__ Row8 load8(const __nv_bfloat16* p) {
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  Row8 r;
  r.v[0] = rbq_bf16lo(u.x); r.v[1] = rbq_bf16hi(u.x); r.v[2] = rbq_bf16lo(u.y); r.v[3] = rbq_bf16hi(u.y);
  r.v[4] = rbq_bf16lo(u.z); r.v[5] = rbq_bf16hi(u.z); r.v[6] = rbq_bf16lo(u.w); r.v[7] = rbq_bf16hi(u.w);
  return r;
}
__device__ __forceinline__ Row8 load8(const float* p) {
  const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  Row8 r;
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}

// exclusive prefix of per-row chunk counts into s_start[0..rows]; every CTA computes the same table
__device__ void build_chunk_table(const int32_t* __restrict__ sel_cnt, const int32_t* __restrict__ n_indexed,
                                  const int32_t* __restrict__ n_total, int rows, int Hq, int* s_start, int* s_warp) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int per = (rows + AT_THREADS - 1) / AT_THREADS;
  const int r0 = tid * per;
  int local = 0;
  for (int r = r0; r < min(rows, r0 + per); ++r) {
    const int b = r / Hq;
    const int na = sel_cnt[r] + max(0, n_total[b] - n_indexed[b]);
    local += (na + AT_CHUNK - 1) / AT_CHUNK;
  }
  int incl = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int woff = 0;
  for (int w = 0; w < warp; ++w) woff += s_warp[w];
  int run = woff + incl - local;
  for (int r = r0; r < min(rows, r0 + per); ++r) {
    const int b = r / Hq;
    const int na = sel_cnt[r] + max(0, n_total[b] - n_indexed[b]);
    s_start[r] = run;
    run += (na + AT_CHUNK - 1) / AT_CHUNK;
  }
  if (tid == AT_THREADS - 1) s_start[rows] = woff + incl;     // rows beyond the last thread's block are empty
  __syncthreads();
  // threads whose block starts beyond `rows` wrote nothing; the last thread holds the grand total
}

template <typename T, typename TQ>
__global__ void __launch_bounds__(AT_THREADS)
attn_chunk_kernel(const TQ* __restrict__ q, const T* __restrict__ K, const T* __restrict__ V, long long sb, long long sh,
                  long long st, const int32_t* __restrict__ sel_idx, const int32_t* __restrict__ sel_cnt,
                  const int32_t* __restrict__ n_indexed, const int32_t* __restrict__ n_total, int rows, int Hq, int Hkv,
                  int Lcap, float sm_scale, float* __restrict__ part, int* __restrict__ chunk_start) {
  __shared__ int s_start[AT_MAX_ROWS + 1];
  __shared__ int s_warp[AT_WARPS];
  __shared__ float s_part[AT_WARPS][AT_PART];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int half = lane >> 4, c = lane & 15;                  // half-warp per row, 8 dims per lane
  const int G = Hq / Hkv;

  build_chunk_table(sel_cnt, n_indexed, n_total, rows, Hq, s_start, s_warp);
  const int total = s_start[rows];
  if (blockIdx.x == 0)
    for (int r = tid; r <= rows; r += AT_THREADS) chunk_start[r] = s_start[r];

  for (int ch = blockIdx.x; ch < total; ch += gridDim.x) {
    // row of this chunk: last r with s_start[r] <= ch
    int lo = 0, hi = rows - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (s_start[mid] <= ch) lo = mid; else hi = mid - 1;
    }
    const int row = lo, b = row / Hq, h = row % Hq, g = h / G;
    const int cnt = sel_cnt[row], nidx = n_indexed[b];
    const int na = cnt + max(0, n_total[b] - nidx);
    const int i0 = (ch - s_start[row]) * AT_CHUNK + warp * 32;   // first item of this warp's strip
    const int nw = max(0, min(32, na - i0));
    const T* Kb = K + (long long)b * sb + (long long)g * sh;
    const T* Vb = V + (long long)b * sb + (long long)g * sh;

    Row8 qv;
    {
      const TQ* qp = q + ((size_t)row * RBQ_D + c * 8);
#pragma unroll
      for (int d = 0; d < 8; ++d) qv.v[d] = rbq_ld_elem(qp, d);
    }
    // this lane's item -> token index
    int my_tok = 0;
    if (lane < nw) {
      const int it = i0 + lane;
      my_tok = (it < cnt) ? sel_idx[(size_t)row * Lcap + it] : nidx + (it - cnt);
    }
    float m = -INFINITY, l = 0.0f, acc[8];
#pragma unroll
    for (int d = 0; d < 8; ++d) acc[d] = 0.0f;

    for (int base = 0; base < nw; base += 8) {
      Row8 kr[4], vr[4];
      bool ok[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int item = base + 2 * j + half;
        const int tok = __shfl_sync(0xffffffffu, my_tok, item & 31);
        ok[j] = item < nw;
        const long long off = (long long)tok * st + c * 8;
        kr[j] = load8(Kb + off);                                // masked items read token 0: harmless
        vr[j] = load8(Vb + off);
      }
      float s[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        float d0 = 0.0f;
#pragma unroll
        for (int d = 0; d < 8; ++d) d0 = fmaf(qv.v[d], kr[j].v[d], d0);
        s[j] = d0;
      }
#pragma unroll
      for (int o = 8; o > 0; o >>= 1)
#pragma unroll
        for (int j = 0; j < 4; ++j) s[j] += __shfl_xor_sync(0xffffffffu, s[j], o);
      float gmax = -INFINITY;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        s[j] = ok[j] ? s[j] * sm_scale : -INFINITY;
        gmax = fmaxf(gmax, s[j]);
      }
      gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, 16));
      const float m_new = fmaxf(m, gmax);                        // finite: item `base` is always valid
      const float resc = __expf(m - m_new);                      // m = -inf -> 0
      l *= resc;
#pragma unroll
      for (int d = 0; d < 8; ++d) acc[d] *= resc;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float p = __expf(s[j] - m_new);                    // masked: exp(-inf) = 0
        l += p;
#pragma unroll
        for (int d = 0; d < 8; ++d) acc[d] = fmaf(p, vr[j].v[d], acc[d]);
      }
      m = m_new;
    }
    // merge the two half-warps (same m), then the warps of the CTA
    l += __shfl_xor_sync(0xffffffffu, l, 16);
#pragma unroll
    for (int d = 0; d < 8; ++d) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], 16);
    if (half == 0) {
#pragma unroll
      for (int d = 0; d < 8; ++d) s_part[warp][c * 8 + d] = acc[d];
      if (c == 0) { s_part[warp][RBQ_D] = m; s_part[warp][RBQ_D + 1] = l; }
    }
    __syncthreads();
    if (tid < RBQ_D) {
      float mm = -INFINITY;
#pragma unroll
      for (int w = 0; w < AT_WARPS; ++w) mm = fmaxf(mm, s_part[w][RBQ_D]);
      float o = 0.0f, ll = 0.0f;
#pragma unroll
      for (int w = 0; w < AT_WARPS; ++w) {
        const float mw = s_part[w][RBQ_D];
        const float f = (mw == -INFINITY) ? 0.0f : __expf(mw - mm);
        o = fmaf(f, s_part[w][tid], o);
        ll = fmaf(f, s_part[w][RBQ_D + 1], ll);
      }
      float* dst = part + (size_t)ch * AT_PART;
      dst[tid] = o;
      if (tid == 0) { dst[RBQ_D] = mm; dst[RBQ_D + 1] = ll; }
    }
    __syncthreads();
  }
}

template <typename TO>
__global__ void __launch_bounds__(RBQ_D)
attn_merge_kernel(const float* __restrict__ part, const int* __restrict__ chunk_start, TO* __restrict__ out,
                  float* __restrict__ lse) {
  const int row = blockIdx.x, d = threadIdx.x;
  const int c0 = chunk_start[row], c1 = chunk_start[row + 1];
  float mm = -INFINITY;
  for (int ch = c0; ch < c1; ++ch) mm = fmaxf(mm, part[(size_t)ch * AT_PART + RBQ_D]);
  float o = 0.0f, l = 0.0f;
  for (int ch = c0; ch < c1; ++ch) {
    const float* p = part + (size_t)ch * AT_PART;
    const float f = (p[RBQ_D] == -INFINITY) ? 0.0f : __expf(p[RBQ_D] - mm);
    o = fmaf(f, p[d], o);
    l = fmaf(f, p[RBQ_D + 1], l);
  }
  const bool empty = !(l > 0.0f);
  rbq_st_elem(out, (long long)row * RBQ_D + d, empty ? 0.0f : o / l);
  if (lse && d == 0) lse[row] = empty ? -INFINITY : mm + logf(l);
}

template <typename T, typename TQ>
int launch_chunks(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const int32_t* sel_idx,
                  const int32_t* sel_cnt, float* part, int* chunk_start, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int grid = ctx->sm_count * 4;
  attn_chunk_kernel<T, TQ><<<grid, AT_THREADS, 0, s>>>((const TQ*)q, (const T*)kv.k, (const T*)kv.v, kv.sb, kv.sh, kv.st,
                                                       sel_idx, sel_cnt, idx->n_indexed, idx->n_total, rows,
                                                       ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads, ctx->cfg.max_tokens,
                                                       ctx->sm_scale, part, chunk_start);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

}  // namespace

int rbq_launch_attention(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const int32_t* sel_idx,
                         const int32_t* sel_cnt, void* out, float* lse, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  if (rows > AT_MAX_ROWS) RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "batch*n_q_heads %d > %d", rows, AT_MAX_ROWS);
  float* part = reinterpret_cast<float*>(static_cast<char*>(ctx->ws) + ctx->off_part);
  int* chunk_start = reinterpret_cast<int*>(static_cast<char*>(ctx->ws) + ctx->off_part_meta);
  const bool kbf = ctx->cfg.kv_dtype == RBQ_BF16, qbf = ctx->cfg.q_dtype == RBQ_BF16;
  int rc;
  if (kbf && qbf) rc = launch_chunks<__nv_bfloat16, __nv_bfloat16>(ctx, q, kv, idx, sel_idx, sel_cnt, part, chunk_start, s);
  else if (kbf) rc = launch_chunks<__nv_bfloat16, float>(ctx, q, kv, idx, sel_idx, sel_cnt, part, chunk_start, s);
  else if (qbf) rc = launch_chunks<float, __nv_bfloat16>(ctx, q, kv, idx, sel_idx, sel_cnt, part, chunk_start, s);
  else rc = launch_chunks<float, float>(ctx, q, kv, idx, sel_idx, sel_cnt, part, chunk_start, s);
  if (rc != RBQ_OK) return rc;
  if (ctx->stage_ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ctx->stage_ev[4], s));
  if (ctx->cfg.out_dtype == RBQ_BF16)
    attn_merge_kernel<<<rows, RBQ_D, 0, s>>>(part, chunk_start, (__nv_bfloat16*)out, lse);
  else
    attn_merge_kernel<<<rows, RBQ_D, 0, s>>>(part, chunk_start, (float*)out, lse);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
