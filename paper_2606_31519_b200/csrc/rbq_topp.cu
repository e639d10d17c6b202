// rbq_topp.cu -- S6: adaptive Top-p selection over the estimated logits
// (Alg.2 line 12, L184; L201 "the minimum set of indices required to cover the probability
// mass p"; tie-break towards the lowest index, R8; p >= 1 selects everything, R9).
//
// The paper's own operator is Alg.3 (L217-252), a ternary threshold search that re-reads the whole
// row 10-25 times with one CTA per row.  Here one THREAD-BLOCK CLUSTER of 8 CTAs owns a row: every
// CTA keeps its slice of the row resident in shared memory (<= 27 K scores), so the row is read from
// L2/HBM exactly once, and the threshold is found by a monotone radix refinement whose per-bin
// (count, mass) histograms are combined across the cluster through distributed shared memory:
//   level 1 : 32 bins of width 1/2 in u = max - score (atomic-free per-thread histograms),
//   level 2+: 256 bins over the surviving key range [cmin, cmax] of the order-preserving uint32
//             float key, 8 more key bits per level (<= 4 levels), u32 shared atomics with
//             fixed-point (2^-40) masses => order-independent, deterministic sums.
// Result: threshold key v*, mass strictly above it, and r = number of entries equal to v* that are
// still needed; the output is every index with key > v* plus the first r (lowest) indices with
// key == v*, written in ascending index order.  Mass is accumulated in fp64 from fp32 expf weights.
#include <cooperative_groups.h>

#include "rbq_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int TP_CS = 8;            // cluster size (portable maximum)
constexpr int TP_THREADS = 512;
constexpr int TP_WARPS = TP_THREADS / 32;
constexpr int NB1 = 32;             // level-1 bins
constexpr int NBX = 256;            // level-2+ bins
constexpr int XW = 3 * NBX + 16;    // exchange words per buffer
constexpr double FX_ONE = 1099511627776.0;   // 2^40

struct TpShared {
  uint32_t xbuf[2][XW];             // cluster exchange buffers (ping-pong)
  uint32_t cnt[NBX], mlo[NBX], mhi[NBX];
  unsigned long long tot_mass[NBX];
  uint32_t tot_cnt[NBX];
  double red_d[TP_WARPS];
  uint32_t red_u[3][TP_WARPS];
  double b_above, b_T;
  uint32_t b_bx, b_cnt, b_found;
  int warp_gt[TP_WARPS], warp_eq[TP_WARPS], warp_out[TP_WARPS], warp_eq0[TP_WARPS];
};

__device__ __forceinline__ float block_max(float v, TpShared& sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) sh.red_u[0][threadIdx.x >> 5] = __float_as_uint(v);
  __syncthreads();
  float r = __uint_as_float(sh.red_u[0][0]);
  for (int w = 1; w < TP_WARPS; ++w) r = fmaxf(r, __uint_as_float(sh.red_u[0][w]));
  __syncthreads();
  return r;
}

// grid = (TP_CS, rows); cluster = TP_CS CTAs along x.  smem: TpShared | scores slice [s_cap] | hist [NB1][TP_THREADS]
__global__ void __cluster_dims__(TP_CS, 1, 1) __launch_bounds__(TP_THREADS)
topp_kernel(const float* __restrict__ scores, const int32_t* __restrict__ n_indexed, int Hq, int Lcap, float p_f,
            int s_cap, int32_t* __restrict__ sel_idx, int32_t* __restrict__ sel_cnt) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TpShared& sh = *reinterpret_cast<TpShared*>(smem_raw);
  float* sc = reinterpret_cast<float*>(smem_raw + ((sizeof(TpShared) + 15) & ~size_t(15)));
  float* hist = sc + s_cap;                                   // [NB1][TP_THREADS]

  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int row = blockIdx.y, b = row / Hq;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n = n_indexed[b];
  const size_t rbase = (size_t)row * Lcap;
  if (n <= 0) {                                               // uniform over the cluster: nobody syncs
    if (rank == 0 && tid == 0) sel_cnt[row] = 0;
    return;
  }
  const int S = (((n + TP_CS - 1) / TP_CS) + 3) & ~3;
  const int lo = rank * S;
  const int len = max(0, min(n, lo + S) - lo);
  if (p_f >= 1.0f) {                                          // R9: everything
    for (int i = tid; i < len; i += TP_THREADS) sel_idx[rbase + lo + i] = lo + i;
    if (rank == 0 && tid == 0) sel_cnt[row] = n;
    return;
  }
  int par = 0;
  auto publish_sync = [&]() { cluster.sync(); par ^= 1; };   // after writing sh.xbuf[par]
  auto remote = [&](int r, int which) -> const uint32_t* {
    return cluster.map_shared_rank(&sh.xbuf[which][0], r);
  };

  // ---- load the slice, row maximum ---------------------------------------------------------------
  float lmax = -INFINITY;
  {
    const float4* src = reinterpret_cast<const float4*>(scores + rbase + lo);
    const int n4 = len >> 2;
    for (int i = tid; i < n4; i += TP_THREADS) {
      const float4 v = src[i];
      reinterpret_cast<float4*>(sc)[i] = v;
      lmax = fmaxf(fmaxf(lmax, fmaxf(v.x, v.y)), fmaxf(v.z, v.w));
    }
    for (int i = (n4 << 2) + tid; i < len; i += TP_THREADS) {
      const float v = scores[rbase + lo + i];
      sc[i] = v;
      lmax = fmaxf(lmax, v);
    }
  }
  lmax = block_max(lmax, sh);
  if (tid == 0) sh.xbuf[par][0] = __float_as_uint(lmax);
  int which = par;
  publish_sync();
  float m = -INFINITY;
  for (int r = 0; r < TP_CS; ++r) m = fmaxf(m, __uint_as_float(remote(r, which)[0]));

  // ---- level 1: 32 bins of width 1/2 in u = m - s, atomic-free --------------------------------------
  for (int bI = 0; bI < NB1; ++bI) hist[bI * TP_THREADS + tid] = 0.0f;
  for (int i = tid; i < len; i += TP_THREADS) {
    const float s = sc[i];
    const float u = __fsub_rn(m, s);
    const int bI = min(NB1 - 1, (int)__fmul_rn(u, 2.0f));
    hist[bI * TP_THREADS + tid] = __fadd_rn(hist[bI * TP_THREADS + tid], expf(__fsub_rn(s, m)));
  }
  __syncthreads();
  for (int bI = warp; bI < NB1; bI += TP_WARPS) {
    double a = 0.0;
    for (int k = 0; k < TP_THREADS / 32; ++k) a += (double)hist[bI * TP_THREADS + lane + 32 * k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) reinterpret_cast<double*>(&sh.xbuf[par][0])[bI] = a;
  }
  which = par;
  publish_sync();
  if (tid < NB1) {
    double a = 0.0;
    for (int r = 0; r < TP_CS; ++r) a += reinterpret_cast<const double*>(remote(r, which))[tid];
    reinterpret_cast<double*>(sh.tot_mass)[tid] = a;
  }
  __syncthreads();
  if (tid == 0) {
    const double* bm = reinterpret_cast<const double*>(sh.tot_mass);
    double Z = 0.0;
    for (int bI = 0; bI < NB1; ++bI) Z += bm[bI];
    const double T = (double)p_f * Z;
    double cum = 0.0;
    int bx = -1, last = 0;
    for (int bI = 0; bI < NB1; ++bI) {
      if (bm[bI] > 0.0) last = bI;
      if (cum + bm[bI] >= T && bm[bI] > 0.0) { bx = bI; break; }
      cum += bm[bI];
    }
    if (bx < 0) { bx = last; cum -= bm[last]; }
    sh.b_T = T; sh.b_above = cum; sh.b_bx = (uint32_t)bx;
  }
  __syncthreads();
  const double T = sh.b_T;
  double above = sh.b_above;
  const int bx1 = (int)sh.b_bx;

  // ---- key range of the crossing bin ---------------------------------------------------------------
  uint32_t kmin = 0xFFFFFFFFu, kmax = 0u, kc = 0u;
  for (int i = tid; i < len; i += TP_THREADS) {
    const float s = sc[i];
    const int bI = min(NB1 - 1, (int)__fmul_rn(__fsub_rn(m, s), 2.0f));
    if (bI == bx1) { const uint32_t k = rbq_fkey(s); kmin = min(kmin, k); kmax = max(kmax, k); ++kc; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
    kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    kc += __shfl_xor_sync(0xffffffffu, kc, o);
  }
  if (lane == 0) { sh.red_u[0][warp] = kmin; sh.red_u[1][warp] = kmax; sh.red_u[2][warp] = kc; }
  __syncthreads();
  if (tid == 0) {
    uint32_t a = 0xFFFFFFFFu, c = 0u, d = 0u;
    for (int w = 0; w < TP_WARPS; ++w) { a = min(a, sh.red_u[0][w]); c = max(c, sh.red_u[1][w]); d += sh.red_u[2][w]; }
    sh.xbuf[par][0] = a; sh.xbuf[par][1] = c; sh.xbuf[par][2] = d;
  }
  which = par;
  publish_sync();
  uint32_t cmin = 0xFFFFFFFFu, cmax = 0u, ctot = 0u;
  for (int r = 0; r < TP_CS; ++r) {
    const uint32_t* rb = remote(r, which);
    cmin = min(cmin, rb[0]); cmax = max(cmax, rb[1]); ctot += rb[2];
  }

  // ---- levels 2+: 256 bins over [cmin, cmax] ---------------------------------------------------------
  uint32_t vstar = cmin, ceq = ctot;
  for (int level = 0; level < 6; ++level) {
    if (cmin >= cmax) { vstar = cmin; ceq = ctot; break; }
    const uint32_t range = cmax - cmin;
    const int bits = 32 - __clz(range);
    const int shift = max(0, bits - 8);
    for (int i = tid; i < NBX; i += TP_THREADS) { sh.cnt[i] = 0; sh.mlo[i] = 0; sh.mhi[i] = 0; }
    __syncthreads();
    for (int i = tid; i < len; i += TP_THREADS) {
      const float s = sc[i];
      const uint32_t k = rbq_fkey(s);
      if (k >= cmin && k <= cmax) {
        const uint32_t bI = (k - cmin) >> shift;
        const unsigned long long fx = __double2ull_rn((double)expf(__fsub_rn(s, m)) * FX_ONE);
        atomicAdd(&sh.cnt[bI], 1u);
        const uint32_t l32 = (uint32_t)fx;
        const uint32_t old = atomicAdd(&sh.mlo[bI], l32);
        const uint32_t carry = (old + l32 < old) ? 1u : 0u;
        const uint32_t h32 = (uint32_t)(fx >> 32) + carry;
        if (h32) atomicAdd(&sh.mhi[bI], h32);
      }
    }
    __syncthreads();
    for (int i = tid; i < NBX; i += TP_THREADS) {
      sh.xbuf[par][i] = sh.cnt[i]; sh.xbuf[par][NBX + i] = sh.mlo[i]; sh.xbuf[par][2 * NBX + i] = sh.mhi[i];
    }
    which = par;
    publish_sync();
    if (tid < NBX) {
      uint32_t c = 0;
      unsigned long long ms = 0;
      for (int r = 0; r < TP_CS; ++r) {
        const uint32_t* rb = remote(r, which);
        c += rb[tid];
        ms += ((unsigned long long)rb[2 * NBX + tid] << 32) + (unsigned long long)rb[NBX + tid];
      }
      sh.tot_cnt[tid] = c; sh.tot_mass[tid] = ms;
    }
    __syncthreads();
    if (warp == 0) {
      // lane l owns bins 255-8l .. 248-8l (descending score order)
      double chunk = 0.0;
      for (int j = 0; j < 8; ++j) chunk += (double)sh.tot_mass[NBX - 1 - 8 * lane - j] * (1.0 / FX_ONE);
      double incl = chunk;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const double v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      const double excl = incl - chunk;
      const bool crosses = (above + incl >= T) && (chunk > 0.0);
      const unsigned bal = __ballot_sync(0xffffffffu, crosses);
      if (bal == 0u) {
        if (lane == 0) sh.b_found = 0;
      } else if (lane == __ffs(bal) - 1) {
        double cum = above + excl;
        int bx = -1, last = -1;
        for (int j = 0; j < 8; ++j) {
          const int bI = NBX - 1 - 8 * lane - j;
          if (sh.tot_cnt[bI] == 0) continue;
          const double md = (double)sh.tot_mass[bI] * (1.0 / FX_ONE);
          last = bI;
          if (cum + md >= T) { bx = bI; break; }
          cum += md;
        }
        if (bx < 0) { bx = last; cum -= (double)sh.tot_mass[last] * (1.0 / FX_ONE); }
        sh.b_found = 1; sh.b_bx = (uint32_t)bx; sh.b_above = cum; sh.b_cnt = sh.tot_cnt[bx];
      }
    }
    __syncthreads();
    if (!sh.b_found) {                                        // rounding: mass ran out -> lowest non-empty bin
      if (tid == 0) {
        double cum = above;
        int last = 0;
        for (int bI = NBX - 1; bI >= 0; --bI) if (sh.tot_cnt[bI]) last = bI;
        for (int bI = NBX - 1; bI > last; --bI) cum += (double)sh.tot_mass[bI] * (1.0 / FX_ONE);
        sh.b_bx = (uint32_t)last; sh.b_above = cum; sh.b_cnt = sh.tot_cnt[last];
      }
      __syncthreads();
    }
    above = sh.b_above;
    const uint32_t bx = sh.b_bx;
    ctot = sh.b_cnt;
    const unsigned long long nmin = (unsigned long long)cmin + ((unsigned long long)bx << shift);
    const unsigned long long nmax = nmin + ((1ull << shift) - 1ull);
    cmin = (uint32_t)nmin;
    cmax = (uint32_t)min(nmax, (unsigned long long)cmax);
    vstar = cmin; ceq = ctot;
    __syncthreads();                                          // sh.b_* reused next level
    if (shift == 0) break;
  }

  // ---- r = entries equal to v* still needed ----------------------------------------------------------
  const double wstar = (double)expf(__fsub_rn(rbq_fkey_inv(vstar), m));
  long long need = 1;
  if (wstar > 0.0) {
    const double x = ceil((T - above) / wstar);
    need = (x < 1.0) ? 1 : (x > (double)ceq ? (long long)ceq : (long long)x);
    while (need > 1 && above + (double)(need - 1) * wstar >= T) --need;       // minimality guard
    while (need < (long long)ceq && above + (double)need * wstar < T) ++need;
  } else {
    need = ceq;
  }

  // ---- ordered selection: key > v*, plus the first `need` indices with key == v* ---------------------
  const int seg = (len + TP_WARPS - 1) / TP_WARPS;            // contiguous warp segments
  const int w0 = min(len, warp * seg), w1 = min(len, w0 + seg);
  int ngt = 0, neq = 0;
  for (int i = w0 + lane; i < w1; i += 32) {
    const uint32_t k = rbq_fkey(sc[i]);
    ngt += (k > vstar); neq += (k == vstar);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { ngt += __shfl_xor_sync(0xffffffffu, ngt, o); neq += __shfl_xor_sync(0xffffffffu, neq, o); }
  if (lane == 0) { sh.warp_gt[warp] = ngt; sh.warp_eq[warp] = neq; }
  __syncthreads();
  if (tid == 0) {
    int g = 0, e = 0;
    for (int w = 0; w < TP_WARPS; ++w) { g += sh.warp_gt[w]; e += sh.warp_eq[w]; }
    sh.xbuf[par][0] = (uint32_t)g; sh.xbuf[par][1] = (uint32_t)e;
  }
  which = par;
  publish_sync();
  long long eq_before = 0, out_base = 0, total = 0;
  {
    long long eqc = 0;
    for (int r = 0; r < TP_CS; ++r) {
      const uint32_t* rb = remote(r, which);
      const long long g = rb[0], e = rb[1];
      const long long take = max(0ll, min(e, need - eqc));
      if (r == rank) { eq_before = eqc; out_base = total; }
      total += g + take;
      eqc += e;
    }
  }
  const long long take_local = max(0ll, min((long long)0x7fffffff, need - eq_before));   // equals this CTA may take
  if (tid == 0) {
    int o = 0, e = 0;
    for (int w = 0; w < TP_WARPS; ++w) {
      sh.warp_out[w] = o; sh.warp_eq0[w] = e;
      const long long tk = max(0ll, min((long long)sh.warp_eq[w], take_local - e));
      o += sh.warp_gt[w] + (int)tk;
      e += sh.warp_eq[w];
    }
  }
  __syncthreads();
  {
    int run_out = sh.warp_out[warp], run_eq = sh.warp_eq0[warp];
    const unsigned lt = (1u << lane) - 1u;
    for (int i0 = w0; i0 < w1; i0 += 32) {
      const int i = i0 + lane;
      uint32_t k = 0;
      const bool valid = i < w1;
      if (valid) k = rbq_fkey(sc[i]);
      const bool isgt = valid && k > vstar, iseq = valid && k == vstar;
      const unsigned beq = __ballot_sync(0xffffffffu, iseq);
      const long long eqr = run_eq + __popc(beq & lt);
      const bool sel = isgt || (iseq && eqr < take_local);
      const unsigned bsel = __ballot_sync(0xffffffffu, sel);
      if (sel) sel_idx[rbase + out_base + run_out + __popc(bsel & lt)] = lo + i;
      run_out += __popc(bsel); run_eq += __popc(beq);
    }
  }
  if (rank == 0 && tid == 0) sel_cnt[row] = (int32_t)total;
  cluster.sync();                                             // keep smem alive until every peer has read it
}

}  // namespace

int rbq_launch_topp(rbq_ctx* ctx, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx,
                    int32_t* sel_cnt, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int s_cap = ((((ctx->cfg.max_tokens + TP_CS - 1) / TP_CS) + 3) & ~3) + 4;
  const size_t smem = ((sizeof(TpShared) + 15) & ~size_t(15)) + (size_t)s_cap * 4 + (size_t)NB1 * TP_THREADS * 4;
  if (smem > 227 * 1024)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select: max_tokens %d exceeds the cluster-resident limit", ctx->cfg.max_tokens);
  static bool attr_set = false;
  if (!attr_set) {
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(topp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    attr_set = true;
  }
  dim3 grid(TP_CS, rows);
  topp_kernel<<<grid, TP_THREADS, smem, s>>>(scores, n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, p, s_cap,
                                             sel_idx, sel_cnt);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
