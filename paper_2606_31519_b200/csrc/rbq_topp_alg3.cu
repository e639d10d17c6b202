// rbq_topp_alg3.cu -- the paper's own Top-p operator: Algorithm 3 "Top-p Mask Generation Logic" (PAPER.md:L217-252,
// 4.1 L256-264, App. B.1), as an alternative selector to the radix select of rbq_topp.cu.
//
// Alg.3 searches a probability threshold by ternary partitioning: per iteration two pivots pi0 < pi1 inside [low, high],
// the masses G0 / G1 above them, and the data-dependent bounds v_min = min{s > low}, v_max = max{s <= high}; it stops
// when v_min = v_max and returns M = (S > low).  The listing lost an `else` between L242 and L245 and initialises low
// with 0 while the text says "min/max" (R12): the restored listing of SURVEY.md Appendix A is used.
//
// B200 design: the paper's kernel (one thread block per row, re-reading the probabilities from global memory in every
// iteration) becomes one 8-CTA thread-block cluster per row with the row RESIDENT in shared memory as fp64 probabilities
// (<= 16 K per CTA); per iteration every thread scans its elements in registers, warps reduce by shuffles, the CTA partial
// goes to all 8 CTAs through distributed shared memory and one cluster barrier ends the iteration; every CTA sums the 8
// partials in rank order, so all take the same branch.  Probabilities and masses are fp64 (the oracle's precision).
// Output: ascending index list + count per row (as rbq_topp_select), optional iteration count.
#include "rbq_common.cuh"
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace {

constexpr int A3_CS = 8;
constexpr int A3_THREADS = 512;
constexpr int A3_WARPS = A3_THREADS / 32;
constexpr int A3_MAX_IT = 4096;

struct A3Part { double g0, g1, vmin, vmax; };

__device__ __forceinline__ A3Part a3_combine(const A3Part& a, const A3Part& b) {
  return {a.g0 + b.g0, a.g1 + b.g1, fmin(a.vmin, b.vmin), fmax(a.vmax, b.vmax)};
}
__device__ __forceinline__ A3Part a3_warp_reduce(A3Part v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    A3Part w;
    w.g0 = __shfl_xor_sync(0xffffffffu, v.g0, o);
    w.g1 = __shfl_xor_sync(0xffffffffu, v.g1, o);
    w.vmin = __shfl_xor_sync(0xffffffffu, v.vmin, o);
    w.vmax = __shfl_xor_sync(0xffffffffu, v.vmax, o);
    v = a3_combine(v, w);
  }
  return v;
}

// grid = (8, rows), cluster (8, 1, 1).  Dynamic shared memory: s_cap doubles (this CTA's slice of the row).
__global__ void __cluster_dims__(A3_CS, 1, 1) __launch_bounds__(A3_THREADS, 1)
topp_alg3_kernel(const float* __restrict__ scores, const int32_t* __restrict__ n_indexed, int Hq, int Lcap, double p,
                 int32_t* __restrict__ sel_idx, int32_t* __restrict__ sel_cnt, int32_t* __restrict__ iters) {
  extern __shared__ __align__(16) unsigned char a3_smem[];
  double* s_prob = reinterpret_cast<double*>(a3_smem);
  __shared__ A3Part s_warp[A3_WARPS];
  __shared__ A3Part s_slot[2][A3_CS];                          // [iteration parity][source rank], written through DSMEM
  __shared__ double s_x[2][A3_CS];                             // set-up exchanges (row maximum, normaliser) and counts
  __shared__ int s_wcnt[A3_WARPS];
  __shared__ int s_ccnt[2 * A3_THREADS];                       // per 32-token chunk: count, then exclusive prefix

  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int row = blockIdx.y, b = row / Hq;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = max(0, min(n_indexed[b], Lcap));
  const int slice = (((n + A3_CS - 1) / A3_CS) + 31) & ~31;    // tokens per CTA (multiple of 32)
  const int t0 = min(n, rank * slice), t1 = min(n, t0 + slice), cnt = t1 - t0;
  const float* srow = scores + (size_t)row * Lcap;

  // all-CTA sum / max of one double per CTA: every CTA writes its value into slot [which][rank] of every CTA
  auto exchange = [&](int which, double v) {
    if (tid < A3_CS) *cluster.map_shared_rank(&s_x[which][rank], tid) = v;
    cluster.sync();
  };
  auto block_reduce = [&](double v, bool is_max) -> double {   // result valid in every thread
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double w = __shfl_xor_sync(0xffffffffu, v, o);
      v = is_max ? fmax(v, w) : v + w;
    }
    __syncthreads();
    if (lane == 0) s_warp[warp].g0 = v;
    __syncthreads();
    double r = s_warp[0].g0;
    for (int w = 1; w < A3_WARPS; ++w) r = is_max ? fmax(r, s_warp[w].g0) : r + s_warp[w].g0;
    return r;
  };

  // ---- probabilities: prob_t = exp(s_t - m) / Z over t < n, fp64 ----------------------------------------------------
  double m_loc = -INFINITY;
  for (int i = tid; i < cnt; i += A3_THREADS) m_loc = fmax(m_loc, (double)srow[t0 + i]);
  exchange(0, block_reduce(m_loc, true));
  double m = -INFINITY;
  for (int r = 0; r < A3_CS; ++r) m = fmax(m, s_x[0][r]);
  double z_loc = 0.0;
  for (int i = tid; i < cnt; i += A3_THREADS) {
    const double e = exp((double)srow[t0 + i] - m);
    s_prob[i] = e;
    z_loc += e;
  }
  exchange(1, block_reduce(z_loc, false));
  double Z = 0.0;
  for (int r = 0; r < A3_CS; ++r) Z += s_x[1][r];
  for (int i = tid; i < cnt; i += A3_THREADS) s_prob[i] = s_prob[i] / Z;
  __syncthreads();

  // ---- Alg.3 lines 3-19 ------------------------------------------------------------------------------------------------
  double low = 0.0, high = 1.0 / Z;                            // max(S): the maximum logit has e = 1
  int it = 0;
  if (n > 0 && p < 1.0) {
    for (;;) {
      ++it;
      const double pi0 = (high + 2.0 * low) / 3.0, pi1 = (2.0 * high + low) / 3.0;
      A3Part a = {0.0, 0.0, INFINITY, -INFINITY};
#pragma unroll 4
      for (int i = tid; i < cnt; i += A3_THREADS) {
        const double s = s_prob[i];
        if (s > pi0) a.g0 += s;
        if (s > pi1) a.g1 += s;
        if (s > low) a.vmin = fmin(a.vmin, s);
        if (s <= high) a.vmax = fmax(a.vmax, s);
      }
      a = a3_warp_reduce(a);
      if (lane == 0) s_warp[warp] = a;
      __syncthreads();
      if (tid < A3_CS) {
        A3Part c = s_warp[0];
        for (int w = 1; w < A3_WARPS; ++w) c = a3_combine(c, s_warp[w]);
        *cluster.map_shared_rank(&s_slot[it & 1][rank], tid) = c;
      }
      cluster.sync();
      A3Part tot = s_slot[it & 1][0];
      for (int r = 1; r < A3_CS; ++r) tot = a3_combine(tot, s_slot[it & 1][r]);
      if (tot.g1 >= p) low = pi1;
      else if (tot.g0 >= p) { low = pi0; high = fmin(pi1, tot.vmax); }
      else high = fmin(pi0, tot.vmax);
      if (tot.vmin == tot.vmax || it > A3_MAX_IT) break;
    }
  } else {
    low = -1.0;                                                 // p >= 1: every indexed token (R13)
  }

  // ---- M = (S > low) as an ascending index list ------------------------------------------------------------------------
  // 32-token chunks: counts by ballot (warp w owns chunks w, w + 16, ...), block scan over the chunk counts, cluster
  // exchange of the CTA totals, then the same ballots place the indices (coalesced stores).
  const int nchunk = (cnt + 31) >> 5;
  for (int c = warp; c < nchunk; c += A3_WARPS) {
    const int i = c * 32 + lane;
    const unsigned bal = __ballot_sync(0xffffffffu, i < cnt && s_prob[i] > low);
    if (lane == 0) s_ccnt[c] = __popc(bal);
  }
  __syncthreads();
  int cta_cnt;
  {
    const int a0 = (2 * tid < nchunk) ? s_ccnt[2 * tid] : 0, a1 = (2 * tid + 1 < nchunk) ? s_ccnt[2 * tid + 1] : 0;
    const int sum = a0 + a1;
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) s_wcnt[warp] = incl;
    __syncthreads();
    int woff = 0, tot = 0;
    for (int w = 0; w < A3_WARPS; ++w) { if (w < warp) woff += s_wcnt[w]; tot += s_wcnt[w]; }
    const int excl = woff + incl - sum;
    if (2 * tid < nchunk) s_ccnt[2 * tid] = excl;
    if (2 * tid + 1 < nchunk) s_ccnt[2 * tid + 1] = excl + a0;
    cta_cnt = tot;
  }
  exchange(0, (double)cta_cnt);                                 // (its cluster barrier also orders the s_ccnt stores)
  int base = 0, total = 0;
  for (int r = 0; r < A3_CS; ++r) { const int v = (int)s_x[0][r]; if (r < rank) base += v; total += v; }
  int32_t* orow = sel_idx + (size_t)row * Lcap;
  for (int c = warp; c < nchunk; c += A3_WARPS) {
    const int i = c * 32 + lane;
    const bool on = i < cnt && s_prob[i] > low;
    const unsigned bal = __ballot_sync(0xffffffffu, on);
    if (on) orow[base + s_ccnt[c] + __popc(bal & ((1u << lane) - 1u))] = t0 + i;
  }
  if (rank == 0 && tid == 0) { sel_cnt[row] = total; if (iters) iters[row] = it; }
  cluster.sync();                                               // no CTA exits while its shared memory may still be written
}

}  // namespace

int rbq_launch_topp_alg3(rbq_ctx* ctx, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx, int32_t* sel_cnt,
                         int32_t* iters, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int s_cap = ((((ctx->cfg.max_tokens + A3_CS - 1) / A3_CS) + 31) & ~31);
  const size_t smem = (size_t)s_cap * sizeof(double);
  if (smem > 200 * 1024 || s_cap > 32 * 2 * A3_THREADS)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select_alg3: max_tokens %d exceeds the cluster-resident limit", ctx->cfg.max_tokens);
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_ALG3, topp_alg3_kernel, 200 * 1024);
  topp_alg3_kernel<<<dim3(A3_CS, rows), A3_THREADS, smem, s>>>(scores, n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, (double)p,
                                                              sel_idx, sel_cnt, iters);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
