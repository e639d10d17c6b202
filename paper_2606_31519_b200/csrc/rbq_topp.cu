// rbq_topp.cu -- S6: adaptive Top-p selection over the estimated logits
// (Alg.2 line 12, L184; L201 "the minimum set of indices required to cover the probability
// mass p"; tie-break towards the lowest index, R8; p >= 1 selects everything, R9).
//
// The paper's own operator is Alg.3 (L217-252), a ternary threshold search that re-reads the whole
// row 10-25 times with one CTA per row.  Here one THREAD-BLOCK CLUSTER of CS CTAs owns a row: every
// CTA keeps its slice of the row resident in shared memory, so the row is read from L2/HBM exactly
// once.  The selection is an exact cut in the total order (score descending, index ascending), i.e.
// on the composite key  C(t) = (orderkey(score_t) << 32) | ~t  whose values are all distinct:
//   level 0 : 2048 bins of width 1/64 in u = max - score (monotone in C).  Per bin a packed
//             (count, sum of r) pair, r = exp(-(u - j/64)) in 2^-28 fixed point, so that the bin
//             mass is exp(-j/64) * sum(r): integer sums => order-independent and deterministic.
//             Histograms are combined across the cluster through distributed shared memory; a block
//             scan (fp64) finds the bin where the cumulative mass crosses T = p * Z.
//   candidates (tokens of the crossing bin, a few hundred at 128 K context) are gathered from all CTAs
//             and ranked exactly with integer prefix masses; the cut C* is the first candidate whose
//             inclusive prefix reaches the remaining mass.  If the crossing bin holds more than
//             TP_CAND tokens (heavy ties), it is first narrowed by 11-bit radix levels on C itself.
//   output  : token t is selected  <=>  C(t) >= C*.  Written as a per-row BITMAP (the representation
//             the gather attention consumes), the count, and -- only when the caller asks for it --
//             the ascending index list.
#include <cooperative_groups.h>

#include "rbq_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int TP_THREADS = 512;
constexpr int TP_WARPS = TP_THREADS / 32;
constexpr int TP_NB = 4 * TP_THREADS;          // 2048 bins, 4 per thread in the scans
constexpr int TP_CAND = 1024;                  // candidates ranked exactly
constexpr unsigned FULL = 0xffffffffu;
typedef unsigned long long u64;

struct TpSmall {
  double wt_d[TP_WARPS];
  u64 wt_u[TP_WARPS];
  uint32_t wt_c[TP_WARPS];
  float red_f[TP_WARPS];
  u64 red_lo[TP_WARPS], red_hi[TP_WARPS];
  // results broadcast inside the CTA
  double trem;            // mass still needed inside the candidate range, in units of 2^-28 * exp(-bx/64)
  u64 rx;                 // total r of the candidate range
  u64 lo64, hi64;         // candidate range on C (refinement only)
  u64 cstar;
  uint32_t bx, cntx, cnt_above, found;
  // read by cluster peers
  float x_max;
  u64 x_lo, x_hi;
  uint32_t x_tot;
  uint32_t lcount;
};

constexpr size_t TP_OFF_HIST = (sizeof(TpSmall) + 127) & ~size_t(127);
constexpr size_t TP_OFF_A = TP_OFF_HIST + TP_NB * sizeof(uint2);                 // 24 KB: cand_all | cand_loc
constexpr size_t TP_A_HALF = TP_CAND * 12;                                       // comp u64 + rfix u32
constexpr size_t TP_OFF_SC = TP_OFF_A + 2 * TP_A_HALF;

__device__ __forceinline__ void bin0(float m, float s, int& j, uint32_t& rfix) {
  const float u = __fsub_rn(m, s);
  j = min(TP_NB - 1, __float2int_rz(__fmul_rn(u, 64.0f)));
  const float frac = __fsub_rn(u, __fmul_rn((float)j, 0.015625f));
  rfix = __float2uint_rn(__fmul_rn(expf(-frac), 268435456.0f));
}
__device__ __forceinline__ int bin0_only(float m, float s) {
  return min(TP_NB - 1, __float2int_rz(__fmul_rn(__fsub_rn(m, s), 64.0f)));
}
__device__ __forceinline__ u64 composite(float s, int t) {
  return ((u64)rbq_fkey(s) << 32) | (u64)(~(uint32_t)t);
}
// hist[j] += (count c, mass v): .x = low 32 bits of the mass, .y = (count << 12) | (mass >> 32)
__device__ __forceinline__ void hist_add(uint2* hist, int j, u64 v, uint32_t c) {
  const uint32_t lo = (uint32_t)v;
  const uint32_t old = atomicAdd(&hist[j].x, lo);
  const uint32_t carry = (old + lo < old) ? 1u : 0u;
  atomicAdd(&hist[j].y, (c << 12) + (uint32_t)(v >> 32) + carry);
}

// totals of this thread's 4 bins over the CS histograms of the cluster
template <int CS>
__device__ __forceinline__ void gather_bins(cg::cluster_group& cluster, uint2* hist, int tid, uint32_t (&cnt)[4], u64 (&R)[4]) {
#pragma unroll
  for (int k = 0; k < 4; ++k) { cnt[k] = 0; R[k] = 0; }
#pragma unroll
  for (int r = 0; r < CS; ++r) {
    const uint4* rh = reinterpret_cast<const uint4*>(CS == 1 ? hist : cluster.map_shared_rank(hist, r)) + tid * 2;
    const uint4 a = rh[0], b = rh[1];
    cnt[0] += a.y >> 12; R[0] += ((u64)(a.y & 0xFFFu) << 32) | a.x;
    cnt[1] += a.w >> 12; R[1] += ((u64)(a.w & 0xFFFu) << 32) | a.z;
    cnt[2] += b.y >> 12; R[2] += ((u64)(b.y & 0xFFFu) << 32) | b.x;
    cnt[3] += b.w >> 12; R[3] += ((u64)(b.w & 0xFFFu) << 32) | b.z;
  }
}

// grid = (CS, rows); cluster = CS CTAs along x.
// smem: TpSmall | hist uint2[TP_NB] (later: selection words) | cand_all | cand_loc | scores slice [s_cap]
template <int CS>
__global__ void __cluster_dims__(CS, 1, 1) __launch_bounds__(TP_THREADS, 2)
topp_kernel(const float* __restrict__ scores, const int32_t* __restrict__ n_indexed, int Hq, int Lcap, int wpr, float p_f,
            uint32_t* __restrict__ sel_bits, int32_t* __restrict__ sel_idx, int32_t* __restrict__ sel_cnt) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TpSmall& sh = *reinterpret_cast<TpSmall*>(smem_raw);
  uint2* hist = reinterpret_cast<uint2*>(smem_raw + TP_OFF_HIST);
  uint32_t* selw = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_HIST);          // aliases hist after the candidate sync
  u64* all_comp = reinterpret_cast<u64*>(smem_raw + TP_OFF_A);
  uint32_t* all_rfix = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_A + TP_CAND * 8);
  uint32_t* woff = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_A);             // aliases cand_all after the cut is known
  u64* loc_comp = reinterpret_cast<u64*>(smem_raw + TP_OFF_A + TP_A_HALF);
  uint32_t* loc_rfix = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_A + TP_A_HALF + TP_CAND * 8);
  float* sc = reinterpret_cast<float*>(smem_raw + TP_OFF_SC);

  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (CS == 1) ? 0 : (int)cluster.block_rank();
  const int row = blockIdx.y, b = row / Hq;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n = n_indexed[b];
  const size_t rbase = (size_t)row * Lcap;
  uint32_t* bits_row = sel_bits + (size_t)row * wpr;
  if (n <= 0) {                                               // uniform over the cluster: nobody syncs
    if (rank == 0 && tid == 0) sel_cnt[row] = 0;
    return;
  }
  const int S = (((n + CS - 1) / CS) + 31) & ~31;             // slice length: whole bitmap words per CTA
  const int lo = rank * S;
  const int len = max(0, min(n, lo + S) - lo);
  const int nwords = (len + 31) >> 5;
  if (p_f >= 1.0f) {                                          // R9: everything
    for (int w = tid; w < nwords; w += TP_THREADS) {
      const int rem = len - w * 32;
      bits_row[(lo >> 5) + w] = rem >= 32 ? 0xFFFFFFFFu : ((1u << rem) - 1u);
    }
    if (sel_idx) for (int i = tid; i < len; i += TP_THREADS) sel_idx[rbase + lo + i] = lo + i;
    if (rank == 0 && tid == 0) sel_cnt[row] = n;
    return;
  }
  auto csync = [&]() { if (CS == 1) __syncthreads(); else cluster.sync(); };
  auto peer = [&](int r) -> const TpSmall* { return CS == 1 ? &sh : cluster.map_shared_rank(&sh, r); };

  // ---- load the slice (read once), zero the histogram, row maximum -----------------------------------
  for (int i = tid; i < TP_NB; i += TP_THREADS) hist[i] = make_uint2(0u, 0u);
  float lmax = -INFINITY;
  {
    const float4* src = reinterpret_cast<const float4*>(scores + rbase + lo);
    const int n4 = len >> 2;
    for (int i = tid; i < n4; i += TP_THREADS) {
      float4 v = src[i];
      v.x = __fadd_rn(v.x, 0.0f); v.y = __fadd_rn(v.y, 0.0f); v.z = __fadd_rn(v.z, 0.0f); v.w = __fadd_rn(v.w, 0.0f);   // -0 -> +0
      reinterpret_cast<float4*>(sc)[i] = v;
      lmax = fmaxf(fmaxf(lmax, fmaxf(v.x, v.y)), fmaxf(v.z, v.w));
    }
    for (int i = (n4 << 2) + tid; i < len; i += TP_THREADS) {
      const float v = __fadd_rn(scores[rbase + lo + i], 0.0f);
      sc[i] = v;
      lmax = fmaxf(lmax, v);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lmax = fmaxf(lmax, __shfl_xor_sync(FULL, lmax, o));
  if (lane == 0) sh.red_f[warp] = lmax;
  __syncthreads();
  if (tid == 0) {
    float r = sh.red_f[0];
    for (int w = 1; w < TP_WARPS; ++w) r = fmaxf(r, sh.red_f[w]);
    sh.x_max = r;
  }
  csync();                                                    // S1: x_max of every CTA visible (and hist zeroed)
  float m = -INFINITY;
#pragma unroll
  for (int r = 0; r < CS; ++r) m = fmaxf(m, peer(r)->x_max);

  // ---- level 0: (count, mass) histogram over u = m - s -------------------------------------------------
  {
    uint32_t of_c = 0;                                        // overflow bin kept in registers (can be half the row)
    u64 of_r = 0;
    for (int base = warp * 32; base < len; base += TP_THREADS) {
      const int i = base + lane;
      int j = -1;
      uint32_t rfix = 0;
      if (i < len) bin0(m, sc[i], j, rfix);
      const int j0 = __shfl_sync(FULL, j, 0);
      if (__all_sync(FULL, j == j0)) {                        // whole warp in one bin (ties): one update
        u64 v = rfix;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
        if (lane == 0) {
          if (j0 == TP_NB - 1) { of_c += 32; of_r += v; } else hist_add(hist, j0, v, 32u);
        }
      } else if (j >= 0) {
        if (j == TP_NB - 1) { of_c += 1; of_r += rfix; } else hist_add(hist, j, (u64)rfix, 1u);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { of_c += __shfl_xor_sync(FULL, of_c, o); of_r += __shfl_xor_sync(FULL, of_r, o); }
    if (lane == 0 && of_c) hist_add(hist, TP_NB - 1, of_r, of_c);
  }
  csync();                                                    // S2: histograms complete

  uint32_t cnt[4];
  u64 R[4];
  gather_bins<CS>(cluster, hist, tid, cnt, R);
  {
    double ms[4], tsum = 0.0;
    uint32_t csum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      ms[k] = (double)R[k] * exp(-(double)(4 * tid + k) * 0.015625);
      tsum += ms[k];
      csum += cnt[k];
    }
    double si = tsum;
    uint32_t ci = csum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double v = __shfl_up_sync(FULL, si, o);
      const uint32_t c = __shfl_up_sync(FULL, ci, o);
      if (lane >= o) { si += v; ci += c; }
    }
    if (lane == 31) { sh.wt_d[warp] = si; sh.wt_c[warp] = ci; }
    if (tid == 0) { sh.bx = 0xFFFFFFFFu; sh.found = 0; sh.lcount = 0; }
    __syncthreads();
    double wp = 0.0, Z = 0.0;
    uint32_t wc = 0;
    for (int w = 0; w < TP_WARPS; ++w) {
      if (w == warp) { wp = Z; }
      Z += sh.wt_d[w];
      if (w < warp) wc += sh.wt_c[w];
    }
    const double T = (double)p_f * Z;
    double se = __shfl_up_sync(FULL, si, 1);
    uint32_t ce = __shfl_up_sync(FULL, ci, 1);
    if (lane == 0) { se = 0.0; ce = 0; }
    const double excl = wp + se, incl = wp + si;              // excl of thread t+1 is bit-identical to incl of thread t
    const bool claim = (excl < T) && (incl >= T);
    if (claim) atomicMin(&sh.bx, (uint32_t)(4 * tid));
    __syncthreads();
    if (claim && sh.bx == (uint32_t)(4 * tid)) {
      double c = excl;
      uint32_t cc = wc + ce;
      int kx = -1;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (kx < 0) {
          if (cnt[k] > 0 && c + ms[k] >= T) kx = k;
          else { c += ms[k]; cc += cnt[k]; }
        }
      }
      if (kx < 0) {                                           // rounding: take the last non-empty bin of this thread
        c = excl; cc = wc + ce;
        int last = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) if (cnt[k] > 0) last = k;
#pragma unroll
        for (int k = 0; k < 4; ++k) if (k < last) { c += ms[k]; cc += cnt[k]; }
        kx = last;
      }
      const int bxx = 4 * tid + kx;
      sh.bx = (uint32_t)bxx;
      sh.cntx = cnt[kx];
      sh.cnt_above = cc;
      sh.rx = R[kx];
      const double rem = (T - c) / exp(-(double)bxx * 0.015625);
      sh.trem = fmin(fmax(rem, 0.5), (double)R[kx]);
    }
    __syncthreads();
  }
  const int bx = (int)sh.bx;
  uint32_t cntx = sh.cntx;
  bool use_range = false;

  // ---- heavy ties only: narrow the candidate range by 11-bit radix levels on C --------------------------
  if (cntx > TP_CAND) {
    u64 mn = ~0ull, mx = 0ull;
    for (int i = tid; i < len; i += TP_THREADS) {
      const float s = sc[i];
      if (bin0_only(m, s) == bx) { const u64 c = composite(s, lo + i); mn = min(mn, c); mx = max(mx, c); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { mn = min(mn, __shfl_xor_sync(FULL, mn, o)); mx = max(mx, __shfl_xor_sync(FULL, mx, o)); }
    if (lane == 0) { sh.red_lo[warp] = mn; sh.red_hi[warp] = mx; }
    __syncthreads();
    if (tid == 0) {
      for (int w = 1; w < TP_WARPS; ++w) { mn = min(mn, sh.red_lo[w]); mx = max(mx, sh.red_hi[w]); }
      sh.x_lo = mn; sh.x_hi = mx;
    }
    csync();                                                  // also: every CTA is done reading the level-0 histograms
    u64 lo64 = ~0ull, hi64 = 0ull;
#pragma unroll
    for (int r = 0; r < CS; ++r) { lo64 = min(lo64, peer(r)->x_lo); hi64 = max(hi64, peer(r)->x_hi); }
    use_range = true;
    while (cntx > TP_CAND) {
      const u64 range = hi64 - lo64;
      const int bits = 64 - __clzll((long long)range);
      const int shift = max(0, bits - 11);
      for (int i = tid; i < TP_NB; i += TP_THREADS) hist[i] = make_uint2(0u, 0u);
      __syncthreads();
      for (int base = warp * 32; base < len; base += TP_THREADS) {
        const int i = base + lane;
        int j = -1;
        uint32_t rfix = 0;
        if (i < len) {
          const float s = sc[i];
          const u64 c = composite(s, lo + i);
          if (c >= lo64 && c <= hi64) {
            int j_unused;
            bin0(m, s, j_unused, rfix);
            j = TP_NB - 1 - (int)((c - lo64) >> shift);       // ascending bin = descending C
          }
        }
        const int j0 = __shfl_sync(FULL, j, 0);
        if (j0 >= 0 && __all_sync(FULL, j == j0)) {
          u64 v = rfix;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
          if (lane == 0) hist_add(hist, j0, v, 32u);
        } else if (j >= 0) {
          hist_add(hist, j, (u64)rfix, 1u);
        }
      }
      csync();
      gather_bins<CS>(cluster, hist, tid, cnt, R);
      u64 tsum = R[0] + R[1] + R[2] + R[3];
      uint32_t csum = cnt[0] + cnt[1] + cnt[2] + cnt[3];
      u64 si = tsum;
      uint32_t ci = csum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const u64 v = __shfl_up_sync(FULL, si, o);
        const uint32_t c = __shfl_up_sync(FULL, ci, o);
        if (lane >= o) { si += v; ci += c; }
      }
      const double trem = sh.trem;                            // read before the barrier: the claiming thread rewrites it below
      if (lane == 31) { sh.wt_u[warp] = si; sh.wt_c[warp] = ci; }
      __syncthreads();
      u64 wp = 0;
      uint32_t wc = 0;
      for (int w = 0; w < warp; ++w) { wp += sh.wt_u[w]; wc += sh.wt_c[w]; }
      const u64 excl = wp + si - tsum, incl = wp + si;
      if ((double)excl < trem && (double)incl >= trem) {       // exact integers: exactly one thread
        u64 c = excl;
        uint32_t cc = wc + ci - csum;
        int kx = -1;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (kx < 0) {
            if ((double)(c + R[k]) >= trem) kx = k;
            else { c += R[k]; cc += cnt[k]; }
          }
        }
        if (kx < 0) kx = 3;
        const int bsel = 4 * tid + kx;
        const u64 nmin = lo64 + ((u64)(TP_NB - 1 - bsel) << shift);
        const u64 nmax = (shift >= 64) ? hi64 : nmin + (((u64)1 << shift) - 1ull);
        sh.lo64 = max(nmin, lo64);
        sh.hi64 = min(nmax, hi64);
        sh.cntx = cnt[kx];
        sh.cnt_above += cc;
        sh.rx = R[kx];
        sh.trem = fmin(trem - (double)c, (double)R[kx]);
      }
      csync();                                                // result visible; peers done reading this level's histogram
      lo64 = sh.lo64; hi64 = sh.hi64; cntx = sh.cntx;
      if (shift == 0) break;                                  // one C per bin: a single candidate is left
    }
  }

  // ---- candidates of this CTA -> local list; gather all; exact ranking ------------------------------------
  {
    u64 lo64 = 0, hi64 = 0;
    if (use_range) { lo64 = sh.lo64; hi64 = sh.hi64; }
    for (int i = tid; i < len; i += TP_THREADS) {
      const float s = sc[i];
      bool is;
      u64 c = composite(s, lo + i);
      if (use_range) is = (c >= lo64 && c <= hi64);
      else is = (bin0_only(m, s) == bx);
      if (is) {
        int j_unused;
        uint32_t rfix;
        bin0(m, s, j_unused, rfix);
        const uint32_t slot = atomicAdd(&sh.lcount, 1u);
        if (slot < TP_CAND) { loc_comp[slot] = c; loc_rfix[slot] = rfix; }
      }
    }
  }
  csync();                                                    // S3: candidate lists complete; histograms free
  int ncand = 0;
#pragma unroll
  for (int r = 0; r < CS; ++r) {
    const TpSmall* ps = peer(r);
    const int lc = min((int)ps->lcount, TP_CAND);
    const u64* rc = CS == 1 ? loc_comp : cluster.map_shared_rank(loc_comp, r);
    const uint32_t* rr = CS == 1 ? loc_rfix : cluster.map_shared_rank(loc_rfix, r);
    for (int k = tid; k < lc; k += TP_THREADS) {
      if (ncand + k < TP_CAND) { all_comp[ncand + k] = rc[k]; all_rfix[ncand + k] = rr[k]; }
    }
    ncand = min(TP_CAND, ncand + lc);
  }
  __syncthreads();
  {
    const double trem = sh.trem;
    for (int i = tid; i < ncand; i += TP_THREADS) {
      const u64 ci = all_comp[i];
      u64 P = 0;
      uint32_t rk = 0;
      for (int j = 0; j < ncand; ++j) {
        const bool ge = all_comp[j] >= ci;
        P += ge ? (u64)all_rfix[j] : 0ull;
        rk += ge ? 1u : 0u;
      }
      if ((double)P >= trem && (double)(P - all_rfix[i]) < trem) { sh.cstar = ci; sh.cnt_above += rk; sh.found = 1; }
    }
    __syncthreads();
    if (!sh.found && tid == 0) {                              // rounding at the last ulp: take every candidate
      u64 mn = ~0ull;
      for (int j = 0; j < ncand; ++j) mn = min(mn, all_comp[j]);
      sh.cstar = mn; sh.cnt_above += (uint32_t)ncand;
    }
    __syncthreads();
  }
  const u64 cstar = sh.cstar;
  const uint32_t total_sel = sh.cnt_above;

  // ---- output: bitmap words (always), ascending index list (on request) -----------------------------------
  for (int w = warp; w < nwords; w += TP_WARPS) {
    const int i = w * 32 + lane;
    const bool sel = (i < len) && composite(sc[i], lo + i) >= cstar;
    const unsigned bal = __ballot_sync(FULL, sel);
    if (lane == 0) { bits_row[(lo >> 5) + w] = bal; selw[w] = bal; }
  }
  if (rank == 0 && tid == 0) sel_cnt[row] = (int32_t)total_sel;
  if (sel_idx) {
    __syncthreads();
    // exclusive scan of popc(selw) over the (<= TP_NB) words of the slice, 4 words per thread
    uint32_t pc[4], tsum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int w = 4 * tid + k;
      pc[k] = (w < nwords) ? __popc(selw[w]) : 0u;
      tsum += pc[k];
    }
    uint32_t si = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(FULL, si, o);
      if (lane >= o) si += v;
    }
    if (lane == 31) sh.wt_c[warp] = si;
    __syncthreads();
    uint32_t wp = 0, tot = 0;
    for (int w = 0; w < TP_WARPS; ++w) { if (w < warp) wp += sh.wt_c[w]; tot += sh.wt_c[w]; }
    uint32_t run = wp + si - tsum;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int w = 4 * tid + k;
      if (w < nwords) woff[w] = run;
      run += pc[k];
    }
    if (tid == 0) sh.x_tot = tot;
    csync();                                                  // S4: per-CTA totals visible
    uint32_t obase = 0;
#pragma unroll
    for (int r = 0; r < CS; ++r) if (r < rank) obase += peer(r)->x_tot;
    const unsigned lt = (1u << lane) - 1u;
    for (int w = warp; w < nwords; w += TP_WARPS) {
      const unsigned bal = selw[w];
      if ((bal >> lane) & 1u) sel_idx[rbase + obase + woff[w] + __popc(bal & lt)] = lo + w * 32 + lane;
    }
  }
  csync();                                                    // keep shared memory alive until every peer has read it
}

template <int CS>
int launch_cs(rbq_ctx* ctx, const float* scores, const int32_t* n_indexed, float p, uint32_t* bits, int wpr, int32_t* sel_idx,
              int32_t* sel_cnt, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int s_cap = ((((ctx->cfg.max_tokens + CS - 1) / CS) + 31) & ~31) + 32;
  const size_t smem = TP_OFF_SC + (size_t)s_cap * 4;
  auto kern = topp_kernel<CS>;
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    RBQ_CUDA_OK(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_smem = smem;
  }
  dim3 grid(CS, rows);
  kern<<<grid, TP_THREADS, smem, s>>>(scores, n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, wpr, p, bits, sel_idx, sel_cnt);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

}  // namespace

// Cluster size: 8 CTAs per row while that still fills the GPU at most ~4 times over; fewer (down to 1) for many
// short rows, as long as the slice of a CTA stays <= 16 K scores (two CTAs per SM).
int rbq_topp_cluster_size(const rbq_ctx* ctx) {
  const long long rows = (long long)ctx->cfg.batch * ctx->cfg.n_q_heads;
  int cs = 8;
  while (cs > 1 && rows * cs > 4ll * ctx->sm_count && (ctx->cfg.max_tokens + cs / 2 - 1) / (cs / 2) <= 16384) cs >>= 1;
  return cs;
}

int rbq_launch_topp(rbq_ctx* ctx, const float* scores, const int32_t* n_indexed, float p, uint32_t* sel_bits, int32_t* sel_idx,
                    int32_t* sel_cnt, cudaStream_t s) {
  const int cs = rbq_topp_cluster_size(ctx);
  const int wpr = rbq_words_per_row(ctx);
  const int s_cap = ((((ctx->cfg.max_tokens + cs - 1) / cs) + 31) & ~31) + 32;
  if (TP_OFF_SC + (size_t)s_cap * 4 > 227 * 1024 || s_cap > 32 * TP_NB)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select: max_tokens %d exceeds the cluster-resident limit", ctx->cfg.max_tokens);
  switch (cs) {
    case 8: return launch_cs<8>(ctx, scores, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    case 4: return launch_cs<4>(ctx, scores, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    case 2: return launch_cs<2>(ctx, scores, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    default: return launch_cs<1>(ctx, scores, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
  }
}
