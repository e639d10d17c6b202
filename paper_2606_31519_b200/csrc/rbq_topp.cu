// rbq_topp.cu -- S6: adaptive Top-p selection over the estimated logits
// (Alg.2 line 12, L184; L201 "the minimum set of indices required to cover the probability
// mass p"; tie-break towards the lowest index, R8; p >= 1 selects everything, R9).
//
// The paper's own operator is Alg.3 (L217-252), a ternary threshold search that re-reads the whole
// row 10-25 times with one CTA per row.  Here one THREAD-BLOCK CLUSTER of CS CTAs owns a row: every
// CTA keeps its slice of the row resident in shared memory, so the row is read from L2/HBM exactly
// once.  The selection is an exact cut in the total order (score descending, index ascending), i.e.
// on the composite key  C(t) = (orderkey(score_t) << 32) | ~t  whose values are all distinct.
// The row maximum m comes with the scores (S5 epilogue, or rowmax_kernel for caller-provided scores):
//   pass 1  : the slice is loaded by cp.async (whole slice in flight) and histogrammed: 2048 bins of width 1/128 in
//             u = m - score (monotone in C).  Per bin a (count, sum of r) pair, r = 2^(22 - (128u - j) log2(e)/128) in
//             2^-22 fixed point, so the bin mass is exp(-j/128) * sum(r): integer sums => order-independent, deterministic.
//             The body is branch-free (two unpredicated shared-memory reductions per token; tokens too deep to be
//             selected -- tp_overflow_bin -- are summed in registers): the pass is bound by issue slots, not by the atomics.
//             Only a 64-bin coarse summary (fp64) and then the 32 fine bins of the crossing coarse bin travel
//             through distributed shared memory (DSMEM is ~20 B/clk per SM).
//   pass 2  : ONE more pass over the resident slice classifies every token: bins above the crossing bin are selected (their
//             bitmap words are assembled right away), the tokens of the crossing bin (a few hundred at 128 K context) become
//             candidates; these are gathered from all CTAs in one DSMEM round; every CTA ranks its share of them against all
//             of them with integer prefix masses (8 threads per candidate) and the one thread that finds the cut C*
//             writes it into every CTA of the cluster.  If the crossing bin holds more than TP_CAND tokens (heavy ties),
//             it is first narrowed by cluster-wide radix levels (TP_LOG_NB bits each) on C.
//   (A variant in which the last of a KV group's row clusters also built the group's union list for S7 in its tail was
//   measured and dropped: on 8 x 4 CTAs the expansion took 32 K cycles, the stand-alone plan kernel on 128 CTAs 8 us.)
//   pass 3  : only the CANDIDATES are revisited: candidate t is selected  <=>  C(t) >= C*; its bit is OR-ed into the words.
//             Output: a per-row BITMAP (the representation the gather attention consumes), the count, and -- only when
//             the caller asks for it -- the ascending index list.
#include <cooperative_groups.h>

#include "rbq_common.cuh"

RBQ_PROBE_DECL(topp_probe);

namespace cg = cooperative_groups;

#ifdef RBQ_PROBE
#define TP_STAMP(slot)                                                                                          \
  do {                                                                                                          \
    const unsigned cta_ = blockIdx.y * gridDim.x + blockIdx.x;                                                   \
    if (threadIdx.x == 0 && cta_ < RBQ_PROBE_CTAS) {                                                             \
      topp_probe[cta_ * RBQ_PROBE_SLOTS + (slot)] = (unsigned long long)clock64();                               \
      if ((slot) == 0) { unsigned long long gt_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_)); topp_probe[cta_ * RBQ_PROBE_SLOTS + 15] = gt_; } \
    }                                                                                                           \
  } while (0)
#else
#define TP_STAMP(slot) do {} while (0)
#endif

#ifndef RBQ_TP_LOG_BINS
#define RBQ_TP_LOG_BINS 11
#endif
// exp(-32 k / TP_SCALE), k < TP_NC, then exp(-i / TP_SCALE), i < 32: the bin-edge weights in fp64, computed once on the
// host (rbq_topp_init)
__device__ double g_tp_tab[(1 << RBQ_TP_LOG_BINS) / 32 + 32];

namespace {

#ifndef RBQ_TP_THREADS
#define RBQ_TP_THREADS 1024
#endif
constexpr int TP_THREADS = RBQ_TP_THREADS;     // 512 or 1024
constexpr int TP_WARPS = TP_THREADS / 32;
constexpr int TP_LOG_NB = RBQ_TP_LOG_BINS;     // 11 or 12
constexpr int TP_NB = 1 << TP_LOG_NB;          // fine bins
constexpr int TP_MAXW = 2048;                  // bitmap words of a slice (<= 65 536 scores per CTA)
constexpr int TP_BPT = TP_NB / TP_THREADS;     // bins (and bitmap words) per thread in the scans: 4 or 2
constexpr int TP_NC = TP_NB / 32;              // coarse bins (32 fine bins each)
constexpr int TP_CAND = 1024;                  // candidates gathered per row
constexpr unsigned FULL = 0xffffffffu;
typedef unsigned long long u64;

struct TpSmall {
  u64 wt_u[TP_WARPS];
  uint32_t wt_c[TP_WARPS];
  u64 red_lo[TP_WARPS], red_hi[TP_WARPS];
  double tabA[TP_NC], tabB[32];                // exp(-32 k / TP_SCALE), exp(-i / TP_SCALE)
  // results broadcast inside the CTA
  double trem;            // mass still needed inside the candidate range, in units of 2^-22 * exp(-bx / TP_SCALE)
  u64 lo64, hi64;         // candidate range on C
  u64 cstar;
  uint32_t bx, cntx, cnt_above, found, ksel;
  // read by cluster peers
  double xc_mass[TP_NC];
  uint32_t xc_cnt[TP_NC];
  u64 x_lo, x_hi;
  uint32_t x_tot;
  uint32_t lcount;
};

constexpr size_t TP_OFF_HIST = (sizeof(TpSmall) + 127) & ~size_t(127);
constexpr size_t TP_OFF_A = TP_OFF_HIST + TP_NB * sizeof(uint2);                 // 24 KB: cand_all | cand_loc
constexpr size_t TP_A_HALF = TP_CAND * 12;                                       // comp u64 + rfix u32
constexpr size_t TP_OFF_SELW = TP_OFF_A + 2 * TP_A_HALF;                          // 8 KB: selection words of the slice (<= 2048)
constexpr size_t TP_OFF_SC = TP_OFF_SELW + TP_MAXW * sizeof(uint32_t);

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// Bin width 1 / TP_SCALE in u = m - s (natural-log units).  The bins reach 16 units, past the overflow bin of a 128 K-token
// row at p = 0.9 (14.3 units).  Narrow bins keep the crossing bin small: the all-pairs ranking of its tokens (the
// candidates) is quadratic -- 6.6 K cycles at config 2 with 2048 bins of 1/64, 4.8 K with 2048 of 1/128, 3.6 K with 4096
// of 1/256 (RBQ_TP_LOG_BINS = 12), which however costs more in the set-up and the crossing search than it saves:
// config 2 step 93.7 vs 94.4 us, config 3 316.9 vs 313.2, config 4 270.6 vs 267.8 -- 2048 bins stay.
constexpr float TP_SCALE = (float)(TP_NB / 16);   // 128 or 256
constexpr float TP_FRAC_LOG2E = -1.4426950408889634f / TP_SCALE;
// fine bin j of u and the fixed-point residual weight r = exp(-(u - j/TP_SCALE)) * 2^22 = 2^(22 - (TP_SCALE u - j) log2(e)/TP_SCALE).
// The XU pipe (conversions, MUFU) is the scarce unit of the histogram pass, so floor() and both float <-> int conversions
// are done with the 2^23 magic-number add on the FMA pipe (round-down for the floor); only ex2 remains on the XU pipe.
// 2^-22 is the resolution of ex2.approx itself.
// jof (integer-valued, <= TP_NB - 1) is the row's OVERFLOW bin: it takes every token with u >= jof / TP_SCALE, r relative to its
// lower edge.  Tokens that deep can never be selected (see tp_overflow_bin), so pass 1 sums them in registers.
// t = TP_SCALE u by ONE FMA on ms = TP_SCALE m: rn(128 m - 128 s) = 128 rn(m - s), scaling by a power of two commutes with
// rounding.
__device__ __forceinline__ float tp_t(float ms, float s) { return fmaf(-TP_SCALE, s, ms); }   // >= 0
__device__ __forceinline__ void bin0(float ms_, float s, float jof, int& j, uint32_t& rfix) {
  const float t = tp_t(ms_, s);
  const float jm = __fadd_rd(fminf(t, jof), 8388608.0f);      // 2^23 + min(floor(t), jof), exact
  j = __float_as_int(jm) - 0x4B000000;
  const float f = __fsub_rn(t, __fsub_rn(jm, 8388608.0f));    // exact for j < jof; large in the overflow bin
  rfix = __float_as_uint(__fadd_rn(ex2_approx(fmaf(f, TP_FRAC_LOG2E, 22.0f)), 8388608.0f)) - 0x4B000000u;
}
// Overflow bin of a row of n tokens at mass p: the tokens with u = m - s > c = ln(1.25 n / (1 - p)) have a total mass below
// n exp(-c) = (1 - p) / 1.25 < (1 - p) Z  (Z >= 1: the maximum itself has weight 1), so the row without them still
// covers p: the minimal covering prefix ends above them and none of them is selected.  They only count towards Z, which
// needs no histogram: all bins from ceil(TP_SCALE c) on are one bin.  (Exactness does not rest on this bound -- a crossing inside
// the overflow bin is resolved by the radix levels on C like any crowded bin -- only the cost does.)  At config 2 this keeps
// 4 % .. 89 % of a row's tokens (40 % on average) out of the shared-memory atomics.  The same value in every CTA of the row.
__device__ __forceinline__ float tp_overflow_bin(int n, float p) {
  const float c = TP_SCALE * __logf(1.25f * (float)n / (1.0f - p));
  return fminf(fmaxf(ceilf(c) + 1.0f, TP_SCALE), (float)(TP_NB - 1));
}
__device__ __forceinline__ u64 composite(float s, int t) {
  return ((u64)rbq_fkey(__fadd_rn(s, 0.0f)) << 32) | (u64)(~(uint32_t)t);   // -0 -> +0: one key for equal scores
}
// Histogram = two u32 arrays (all 32 banks in use): hist[j] = low 32 bits of the mass, hist[TP_NB + j] = (count << 12) |
// (mass >> 32).  hist[j] += (count c, mass v):
// (explicit shared-space atomics on a 32-bit shared address: a generic-pointer atomicAdd makes the compiler rebuild the
// shared-window address from SR_CgaCtaId for every atomic inside a cluster kernel)
__device__ __forceinline__ void hist_add(uint32_t hist_sa, int j, u64 v, uint32_t c) {
  const uint32_t sa = hist_sa + 4u * (uint32_t)j;
  const uint32_t lo = (uint32_t)v;
  uint32_t old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(sa), "r"(lo) : "memory");
  const uint32_t carry = (old + lo < old) ? 1u : 0u;
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(sa + 4u * TP_NB), "r"((c << 12) + (uint32_t)(v >> 32) + carry) : "memory");
}
// Pass-1 form of the histogram: two u32 arrays, hist[j] = sum of d = 2^22 - r and hist[TP_NB + j] = count.  Inside a
// bin r lies in (0.989 * 2^22, 2^22], so d < 2^16 and the sums of a CTA's <= 41 K tokens stay below 2^31 (read back as
// signed: ex2.approx may return 2^22 + 1 ulp).  Two reductions without return value, never predicated: a token that is
// not histogrammed (overflow bin, inactive lane) adds to a per-lane dummy word behind the histogram instead (ptxas turns
// predicated shared atomics into branch + reconvergence pairs, ~3 extra issue slots each).  Folded into the
// (lo, count | hi) form after the pass.
__device__ __forceinline__ void hist_add2(uint32_t sa, uint32_t d, uint32_t c) {
  asm volatile("red.shared.add.u32 [%0], %1;\n\tred.shared.add.u32 [%0 + %3], %2;" ::"r"(sa), "r"(d), "r"(c), "n"(4 * TP_NB) : "memory");
}
// Histogram step of pass 1 for the four scores of one float4 group.  A token of the overflow bin (or of an inactive lane:
// d = c = 0) goes to one of TP_OFS per-(warp & 3, lane) slot pairs behind the histogram -- conflict-free, and no register
// bookkeeping: <= 320 tokens per slot, d <= 2^22, so a slot's sum stays below 2^31.  128 tokens in one bin (ties): one pair
// of reductions for the warp.
constexpr int TP_OFS = 128;
template <bool ALL_ACTIVE>
__device__ __forceinline__ void tp_hist4(const float4 t4, bool act, float ms_, float jof_f, int jof, uint32_t hist_sa, uint32_t slot_sa, int lane) {
  const float v[4] = {t4.x, t4.y, t4.z, t4.w};
  int j[4];
  uint32_t rf[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) bin0(ms_, v[k], jof_f, j[k], rf[k]);
  const int j0 = __shfl_sync(FULL, j[0], 0);
  const bool same = (ALL_ACTIVE || act) && j[0] == j0 && j[1] == j0 && j[2] == j0 && j[3] == j0;
  if (__all_sync(FULL, same) && j0 != jof) {
    const uint32_t d = __reduce_add_sync(FULL, (4u << 22) - (rf[0] + rf[1] + rf[2] + rf[3]));
    if (lane == 0) hist_add2(hist_sa + 4u * (uint32_t)j0, d, 128u);
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const bool tobin = (ALL_ACTIVE || act) && j[k] != jof;
      const uint32_t d = (1u << 22) - rf[k];
      hist_add2(tobin ? hist_sa + 4u * (uint32_t)j[k] : slot_sa, (ALL_ACTIVE || act) ? d : 0u, (ALL_ACTIVE || act) ? 1u : 0u);
    }
  }
}
__device__ __forceinline__ void unpack_bin(uint2 v, uint32_t& cnt, u64& R) {
  cnt = v.y >> 12;
  R = ((u64)(v.y & 0xFFFu) << 32) | v.x;
}

// totals of this thread's TP_BPT bins over the CS histograms of the cluster (cluster-wide radix levels only)
template <int CS>
__device__ __forceinline__ void gather_bins(cg::cluster_group& cluster, uint32_t* hist, int tid, uint32_t (&cnt)[TP_BPT], u64 (&R)[TP_BPT]) {
#pragma unroll
  for (int k = 0; k < TP_BPT; ++k) { cnt[k] = 0; R[k] = 0; }
#pragma unroll
  for (int r = 0; r < CS; ++r) {
    const uint32_t* rh = CS == 1 ? hist : cluster.map_shared_rank(hist, r);
#pragma unroll
    for (int k = 0; k < TP_BPT; ++k) {
      uint32_t c; u64 v;
      unpack_bin(make_uint2(rh[TP_BPT * tid + k], rh[TP_NB + TP_BPT * tid + k]), c, v);
      cnt[k] += c; R[k] += v;
    }
  }
}

// Integer block scan over TP_NB bins (TP_BPT per thread, ascending bin = descending C): finds the bin where the inclusive
// prefix of R first reaches sh.trem (clamped to the total), and updates sh.{trem, cnt_above, cntx, lo64, hi64}.
// `lo64`, `hi64`, `shift` describe the binning  bin = TP_NB-1 - ((C - lo64) >> shift).  Ends with a block barrier.
__device__ __forceinline__ void radix_scan(TpSmall& sh, const uint32_t (&cnt)[TP_BPT], const u64 (&R)[TP_BPT], u64 lo64, u64 hi64, int shift) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  u64 tsum = 0;
  uint32_t csum = 0;
#pragma unroll
  for (int k = 0; k < TP_BPT; ++k) { tsum += R[k]; csum += cnt[k]; }
  u64 si = tsum;
  uint32_t ci = csum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const u64 v = __shfl_up_sync(FULL, si, o);
    const uint32_t c = __shfl_up_sync(FULL, ci, o);
    if (lane >= o) { si += v; ci += c; }
  }
  const double trem_in = sh.trem;                               // read before the barrier: the claiming thread rewrites it
  if (lane == 31) { sh.wt_u[warp] = si; sh.wt_c[warp] = ci; }
  __syncthreads();
  if (warp == 0) {                                              // warp totals -> exclusive prefixes + grand total, by one warp (every
    const u64 v = lane < TP_WARPS ? sh.wt_u[lane] : 0ull;        // thread summing the <= 32 totals itself costs ~3 K cycles of shared-
    const uint32_t c = lane < TP_WARPS ? sh.wt_c[lane] : 0u;     // memory loads at 1 024 threads)
    u64 vi = v;
    uint32_t cx = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const u64 v2 = __shfl_up_sync(FULL, vi, o);
      const uint32_t c2 = __shfl_up_sync(FULL, cx, o);
      if (lane >= o) { vi += v2; cx += c2; }
    }
    if (lane < TP_WARPS) { sh.wt_u[lane] = vi - v; sh.wt_c[lane] = cx - c; }
    if (lane == 31) sh.red_lo[0] = vi;
  }
  __syncthreads();
  const u64 wp = sh.wt_u[warp], tot = sh.red_lo[0];
  const uint32_t wc = sh.wt_c[warp];
  const double trem = fmin(trem_in, (double)tot);
  const u64 excl = wp + si - tsum, incl = wp + si;
  // exact integers: exactly one thread claims.  tot == 0 (every candidate weight underflows): first non-empty bin.
  const bool claim = tot > 0 ? ((double)excl < trem && (double)incl >= trem) : (wc + ci - csum == 0 && csum > 0);
  if (claim) {
    u64 c = excl;
    uint32_t cc = wc + ci - csum;
    int kx = -1;
#pragma unroll
    for (int k = 0; k < TP_BPT; ++k) {
      if (kx < 0) {
        if (tot > 0 ? ((double)(c + R[k]) >= trem) : (cnt[k] > 0)) kx = k;
        else { c += R[k]; cc += cnt[k]; }
      }
    }
    if (kx < 0) kx = TP_BPT - 1;
    const int bsel = TP_BPT * tid + kx;
    const u64 nmin = lo64 + ((u64)(TP_NB - 1 - bsel) << shift);
    const u64 nmax = nmin + (((u64)1 << shift) - 1ull);
    sh.lo64 = max(nmin, lo64);
    sh.hi64 = min(nmax, hi64);
    sh.cntx = cnt[kx];
    sh.cnt_above += cc;
    sh.trem = fmin(trem - (double)c, (double)R[kx]);
  }
  __syncthreads();
}

// grid = (CS, rows); cluster = CS CTAs along x.
// smem: TpSmall | hist u32[2][TP_NB] (later: selection words) | cand_all | cand_loc | scores slice [s_cap]
template <int CS>
__global__ void __cluster_dims__(CS, 1, 1) __launch_bounds__(TP_THREADS, TP_THREADS == 512 ? 2 : 1)
topp_kernel(const float* __restrict__ scores, uint32_t* __restrict__ rowmax_key, const int32_t* __restrict__ n_indexed,
            int Hq, int Lcap, int wpr, float p_f, uint32_t* __restrict__ sel_bits, int32_t* __restrict__ sel_idx,
            int32_t* __restrict__ sel_cnt) {
  rbq_pdl_trigger();                                          // (dependents: the gather cannot be resident beside this kernel anyway)
  TP_STAMP(0);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TpSmall& sh = *reinterpret_cast<TpSmall*>(smem_raw);
  uint32_t* hist = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_HIST);
  uint32_t hist_sa = (uint32_t)__cvta_generic_to_shared(hist);   // 32-bit shared address for the histogram atomics,
  asm volatile("mov.u32 %0, %0;" : "+r"(hist_sa));               // opaque: kept in a register, not rebuilt from SR_CgaCtaId per atomic
  uint32_t* selw = reinterpret_cast<uint32_t*>(smem_raw + TP_OFF_SELW);          // own area: written while peers may still read hist
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
    rbq_pdl_wait();
    if (rank == 0 && tid == 0) sel_cnt[row] = 0;
    return;
  }
  const int S = (((n + CS - 1) / CS) + 31) & ~31;             // slice length: whole bitmap words per CTA
  const int lo = rank * S;
  const int len = max(0, min(n, lo + S) - lo);
  const int nwords = (len + 31) >> 5;
  if (p_f >= 1.0f) {                                          // R9: everything
    rbq_pdl_wait();
    for (int w = tid; w < nwords; w += TP_THREADS) {
      const int rem = len - w * 32;
      bits_row[(lo >> 5) + w] = rem >= 32 ? 0xFFFFFFFFu : ((1u << rem) - 1u);
    }
    if (sel_idx) for (int i = tid; i < len; i += TP_THREADS) sel_idx[rbase + lo + i] = lo + i;
    if (rank == 0 && tid == 0) { sel_cnt[row] = n; rowmax_key[row] = 0u; }   // nobody reads the key on this path
    return;
  }
  auto csync = [&]() { if (CS == 1) __syncthreads(); else cluster.sync(); };
  auto peer = [&](int r) -> const TpSmall* { return CS == 1 ? &sh : cluster.map_shared_rank(&sh, r); };

  // ---- pass 1: load the slice (read once) and histogram it ---------------------------------------------
  // A CTA of 1 024 threads x 64 registers becomes resident only when its SM has drained, i.e. at the very end of S5: the
  // set-up below is not hidden behind the predecessor.  So the wait comes first, the slice copies go out right behind it and
  // the histogram is zeroed while they are in flight.
  const double tabv = tid < TP_NC + 32 ? g_tp_tab[tid] : 0.0;    // written at rbq_create, not by a kernel of the chain
  rbq_pdl_wait();                                             // scores and row maxima of S5
  TP_STAMP(1);
  const float jof_f = tp_overflow_bin(n, p_f);
  const int jof = (int)jof_f;
  float m, ms_;                                               // row maximum: loaded behind the slice copies (one latency, not two)
  {
    const float4* src = reinterpret_cast<const float4*>(scores + rbase + lo);
    const float4* sc4 = reinterpret_cast<const float4*>(sc);
    const int n4 = (len + 3) >> 2;                            // whole float4 groups (Lcap % 4 == 0: in bounds)
    // the whole slice in flight at once (16-byte cp.async, one latency round), then histogrammed from shared memory.
    // (Committing the rounds in four groups and starting on the first while the rest is in flight was measured: the
    // first group lands when nearly everything has -- no gain.)
    {
      const uint32_t sdst = (uint32_t)__cvta_generic_to_shared(sc);
      for (int i4 = tid; i4 < n4; i4 += TP_THREADS)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sdst + 16u * (uint32_t)i4), "l"(src + i4) : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
      const uint32_t mkey = rowmax_key[row];
      for (int i = tid; i < 2 * TP_NB; i += TP_THREADS) hist[i] = 0u;
      if (tid < TP_OFS) { hist[2 * TP_NB + tid] = 0u; hist[3 * TP_NB + tid] = 0u; }   // overflow slots (candidate area, free until S1)
      if (tid == 0) { sh.lcount = 0; sh.found = 0; }
      __syncthreads();                                         // histogram zeroed by all before anybody adds to it (the copies are still
                                                               // in flight: every thread then starts on its own groups as they land)
      if (tid < TP_NC) sh.tabA[tid] = tabv;                    // fp64 tables: loaded at kernel entry, first used after the pass
      else if (tid < TP_NC + 32) sh.tabB[tid - TP_NC] = tabv;
      m = __fadd_rn(rbq_fkey_inv(mkey), 0.0f);
      ms_ = __fmul_rn(m, TP_SCALE);
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    TP_STAMP(10);
    // Branch-free body over the FULL float4 groups (each thread reads back exactly the groups it copied); whole rounds first,
    // then the last, partial round, whose inactive lanes re-read the last group and add zeros.  The issue slots are the
    // limiter here (measured: dropping atomics changes little; ncu: 'not selected' is the top stall).
    const int n4f = len >> 2;
    const uint32_t slot_sa = hist_sa + 4u * (uint32_t)(2 * TP_NB + (warp & 3) * 32 + lane);   // count slot: + 4 TP_NB
    const int full = n4f & ~(TP_THREADS - 1);
#pragma unroll 2
    for (int i4 = tid; i4 < full; i4 += TP_THREADS) tp_hist4<true>(sc4[i4], true, ms_, jof_f, jof, hist_sa, slot_sa, lane);
    if (full + warp * 32 < n4f) {                              // warp-uniform
      const int i4 = full + tid;
      const bool act = i4 < n4f;
      tp_hist4<false>(sc4[act ? i4 : n4f - 1], act, ms_, jof_f, jof, hist_sa, slot_sa, lane);
    }
    if ((len & 3) && tid == (n4f & (TP_THREADS - 1))) {        // the ragged tail (<= 3 tokens), by the thread that copied it
      for (int k = 0; k < (len & 3); ++k) {
        int j;
        uint32_t rf;
        bin0(ms_, sc[4 * n4f + k], jof_f, j, rf);
        hist_add2(j != jof ? hist_sa + 4u * (uint32_t)j : slot_sa, (1u << 22) - rf, 1u);
      }
    }
  }
  __syncthreads();
  // slice padded to whole bitmap words with -inf (t = +inf: neither selected nor a candidate): pass 2 runs unguarded
  if (tid < nwords * 32 - len) sc[len + tid] = -INFINITY;
  for (int b = tid; b < TP_NB; b += TP_THREADS) {               // fold into hist[b] = mass lo, hist[TP_NB + b] = count << 12 | mass hi
    if (b == jof) continue;                                     // the overflow bin: from its slots, below
    const uint32_t cnt = hist[TP_NB + b];
    const u64 mass = ((u64)cnt << 22) - (u64)(long long)(int)hist[b];
    hist[b] = (uint32_t)mass;
    hist[TP_NB + b] = (cnt << 12) | (uint32_t)(mass >> 32);
  }
  if (warp == 0) {                                              // overflow bin = its own (empty) histogram word + the TP_OFS slots
    uint32_t cnt = 0;
    long long dsum = 0;
#pragma unroll
    for (int k = 0; k < TP_OFS / 32; ++k) {
      cnt += hist[3 * TP_NB + 32 * k + lane];
      dsum += (long long)(int)hist[2 * TP_NB + 32 * k + lane];
    }
    cnt = __reduce_add_sync(FULL, cnt);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dsum += __shfl_xor_sync(FULL, dsum, o);
    if (lane == 0) {
      cnt += hist[TP_NB + jof];
      const u64 mass = ((u64)cnt << 22) - (u64)(dsum + (long long)(int)hist[jof]);
      hist[jof] = (uint32_t)mass;
      hist[TP_NB + jof] = (cnt << 12) | (uint32_t)(mass >> 32);
    }
  }
  __syncthreads();
  // coarse summary of this CTA: 64 bins of 32 fine bins; thread t owns fine bins TP_BPT t .., 32 / TP_BPT threads per coarse bin
  {
    constexpr int TPC = 32 / TP_BPT;
    double ms = 0.0;
    uint32_t cs = 0;
#pragma unroll
    for (int k = 0; k < TP_BPT; ++k) {
      uint32_t c; u64 R;
      unpack_bin(make_uint2(hist[TP_BPT * tid + k], hist[TP_NB + TP_BPT * tid + k]), c, R);
      ms += (double)R * sh.tabB[(TP_BPT * tid + k) & 31];
      cs += c;
    }
#pragma unroll
    for (int o = 1; o < TPC; o <<= 1) { ms += __shfl_xor_sync(FULL, ms, o); cs += __shfl_xor_sync(FULL, cs, o); }
    if ((tid & (TPC - 1)) == 0) { sh.xc_mass[tid / TPC] = ms * sh.tabA[tid / TPC]; sh.xc_cnt[tid / TPC] = cs; }
  }
  TP_STAMP(2);
  csync();                                                    // S1: histograms and coarse summaries complete
  TP_STAMP(3);
  if (rank == 0 && tid == 0) rowmax_key[row] = 0u;            // every CTA of the row has read its maximum: clear the key for the next step
  if (warp == 0) {
    // coarse crossing: lane l owns coarse bins CPL l .. CPL l + CPL - 1 (totals over the cluster in rank order), warp scan
    // in fp64; then the 32 fine bins of the crossing coarse bin, one per lane
    constexpr int CPL = TP_NC / 32;
    double mk[CPL], msum = 0.0;
    uint32_t ck[CPL], csum = 0;
#pragma unroll
    for (int k = 0; k < CPL; ++k) { mk[k] = 0.0; ck[k] = 0; }
#pragma unroll
    for (int r = 0; r < CS; ++r) {
      const TpSmall* ps = peer(r);
#pragma unroll
      for (int k = 0; k < CPL; ++k) { mk[k] += ps->xc_mass[CPL * lane + k]; ck[k] += ps->xc_cnt[CPL * lane + k]; }
    }
#pragma unroll
    for (int k = 0; k < CPL; ++k) { msum += mk[k]; csum += ck[k]; }
    double si2 = msum;
    uint32_t ci2 = csum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double v = __shfl_up_sync(FULL, si2, o);
      const uint32_t cv = __shfl_up_sync(FULL, ci2, o);
      if (lane >= o) { si2 += v; ci2 += cv; }
    }
    const double Z = __shfl_sync(FULL, si2, 31);
    double T = (double)p_f * Z;
    const double ex2 = si2 - msum;
    const uint32_t cex = ci2 - csum;
    int kfirst = -1, klast = 0;                                  // first crossing bin of this lane; its last non-empty bin
    {
      double run = ex2;
#pragma unroll
      for (int k = 0; k < CPL; ++k) {
        if (kfirst < 0 && ck[k] > 0 && run + mk[k] >= T) kfirst = k;
        if (ck[k] > 0) klast = k;
        run += mk[k];
      }
    }
    unsigned cb = __ballot_sync(FULL, kfirst >= 0);
    const unsigned ne = __ballot_sync(FULL, csum != 0);
    bool forced = false;
    if (cb == 0u) { cb = ne ? (1u << (31 - __clz(ne))) : 1u; forced = true; }   // rounding at the last ulp: last non-empty bin
    const int lsel = __ffs(cb) - 1;
    int kx = 0;
    double above = 0.0;
    uint32_t cab = 0;
    if (lane == lsel) {
      const int ks = forced ? klast : kfirst;
      above = ex2;
      cab = cex;
#pragma unroll
      for (int k = 0; k < CPL; ++k) if (k < ks) { above += mk[k]; cab += ck[k]; }
      kx = CPL * lane + ks;
    }
    kx = __shfl_sync(FULL, kx, lsel); above = __shfl_sync(FULL, above, lsel); cab = __shfl_sync(FULL, cab, lsel);
    uint32_t c = 0;
    u64 R = 0;
#pragma unroll
    for (int r = 0; r < CS; ++r) {
      const uint32_t* rh = CS == 1 ? hist : cluster.map_shared_rank(hist, r);
      uint32_t cc; u64 rr;
      unpack_bin(make_uint2(rh[32 * kx + lane], rh[TP_NB + 32 * kx + lane]), cc, rr);
      c += cc; R += rr;
    }
    const double e = sh.tabA[kx] * sh.tabB[lane];
    const double ms = (double)R * e;
    double si = ms;
    uint32_t ci = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double v = __shfl_up_sync(FULL, si, o);
      const uint32_t cv = __shfl_up_sync(FULL, ci, o);
      if (lane >= o) { si += v; ci += cv; }
    }
    const bool cross = c > 0 && above + si >= T;
    unsigned bal = __ballot_sync(FULL, cross);
    const unsigned nonempty = __ballot_sync(FULL, c > 0);
    if (bal == 0u) bal = nonempty ? (1u << (31 - __clz(nonempty))) : 1u;      // rounding at the last ulp: last non-empty bin
    const int lx = __ffs(bal) - 1;
    if (lane == lx) {
      const double ab = above + (si - ms);
      sh.bx = (uint32_t)(32 * kx + lane);
      sh.cntx = c;
      sh.cnt_above = cab + (ci - c);
      sh.trem = fmin(fmax((T - ab) / e, 0.5), (double)R);
    }
  }
  __syncthreads();
  TP_STAMP(4);
  const int bx = (int)sh.bx;
  uint32_t cntx = sh.cntx;
  const float t_lo = (float)bx, t_hi = (bx == jof) ? INFINITY : (float)(bx + 1);   // the crossing bin in t = TP_SCALE u
  bool use_range = false;

  // ---- heavy ties only: narrow the candidate range by cluster-wide 11-bit radix levels on C --------------
  if (cntx > TP_CAND) {
    u64 mn = ~0ull, mx = 0ull;
    for (int i = tid; i < len; i += TP_THREADS) {
      const float s = sc[i];
      const float t = tp_t(ms_, s);
      if (t >= t_lo && t < t_hi) { const u64 c = composite(s, lo + i); mn = min(mn, c); mx = max(mx, c); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { mn = min(mn, __shfl_xor_sync(FULL, mn, o)); mx = max(mx, __shfl_xor_sync(FULL, mx, o)); }
    if (lane == 0) { sh.red_lo[warp] = mn; sh.red_hi[warp] = mx; }
    __syncthreads();
    if (tid == 0) {
      for (int w = 1; w < TP_WARPS; ++w) { mn = min(mn, sh.red_lo[w]); mx = max(mx, sh.red_hi[w]); }
      sh.x_lo = mn; sh.x_hi = mx;
    }
    csync();                                                  // also: every CTA is done reading the pass-1 histograms
    u64 lo64 = ~0ull, hi64 = 0ull;
#pragma unroll
    for (int r = 0; r < CS; ++r) { lo64 = min(lo64, peer(r)->x_lo); hi64 = max(hi64, peer(r)->x_hi); }
    use_range = true;
    while (cntx > TP_CAND) {
      const u64 range = hi64 - lo64;
      const int shift = max(0, (64 - __clzll((long long)range)) - TP_LOG_NB);
      for (int i = tid; i < 2 * TP_NB; i += TP_THREADS) hist[i] = 0u;
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
            bin0(ms_, s, jof_f, j_unused, rfix);
            j = TP_NB - 1 - (int)((c - lo64) >> shift);       // ascending bin = descending C
          }
        }
        const int j0 = __shfl_sync(FULL, j, 0);
        if (j0 >= 0 && __all_sync(FULL, j == j0)) {
          u64 v = rfix;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
          if (lane == 0) hist_add(hist_sa, j0, v, 32u);
        } else if (j >= 0) {
          hist_add(hist_sa, j, (u64)rfix, 1u);
        }
      }
      csync();
      uint32_t cnt[TP_BPT];
      u64 R[TP_BPT];
      gather_bins<CS>(cluster, hist, tid, cnt, R);
      radix_scan(sh, cnt, R, lo64, hi64, shift);
      csync();                                                // peers done reading this level's histogram
      lo64 = sh.lo64; hi64 = sh.hi64; cntx = sh.cntx;
      if (shift == 0) break;                                  // one C per bin: a single candidate is left
    }
  }

  // ---- pass 2: every token classified once: above the crossing bin -> its bit (8 lanes assemble one 32-token word);
  //      in the crossing bin (and, after a radix narrowing, inside the candidate range) -> local candidate list.
  //      Unguarded and branch-free over whole words (the pad is -inf); the candidates (a few hundred per row) take a
  //      warp-uniform side branch ----------
  {
    u64 lo64 = 0, hi64 = 0;
    if (use_range) { lo64 = sh.lo64; hi64 = sh.hi64; }
    const float4* sc4 = reinterpret_cast<const float4*>(sc);
    const int n4r = nwords * 8;                               // float4 groups of whole words
#pragma unroll 2
    for (int base = warp * 32; base < n4r; base += TP_THREADS) {
      const int i4 = base + lane;
      const bool act = i4 < n4r;
      const float4 v4 = sc4[act ? i4 : n4r - 1];
      const float v[4] = {v4.x, v4.y, v4.z, v4.w};
      uint32_t nib = 0, cm = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float t = tp_t(ms_, v[k]);
        nib |= (t < t_lo) ? (1u << k) : 0u;
        cm |= (t >= t_lo && t < t_hi) ? (1u << k) : 0u;
      }
      if (!act) cm = 0;
      if (__any_sync(FULL, cm != 0)) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (cm & (1u << k)) {
            const u64 c = composite(v[k], lo + 4 * i4 + k);
            if (!use_range || (c >= lo64 && c <= hi64)) {
              int j_unused;
              uint32_t rfix;
              bin0(ms_, v[k], jof_f, j_unused, rfix);
              const uint32_t slot = atomicAdd(&sh.lcount, 1u);
              if (slot < TP_CAND) { loc_comp[slot] = c; loc_rfix[slot] = rfix; }
            } else if (c > hi64) {
              nib |= 1u << k;                                 // narrowed range: above it = selected for sure
            }
          }
        }
      }
      uint32_t word = nib << (4 * (lane & 7));
      word |= __shfl_xor_sync(FULL, word, 1);
      word |= __shfl_xor_sync(FULL, word, 2);
      word |= __shfl_xor_sync(FULL, word, 4);
      if ((lane & 7) == 0 && act) selw[i4 >> 3] = word;
    }
  }
  TP_STAMP(5);
  csync();                                                    // S2: candidate lists complete; histograms free
  TP_STAMP(6);
  int ncand = 0;
  {
    int off[CS + 1];                                          // all peer counts first, then one round of independent remote loads
    off[0] = 0;
#pragma unroll
    for (int r = 0; r < CS; ++r) off[r + 1] = min(TP_CAND, off[r] + min((int)peer(r)->lcount, TP_CAND));
    ncand = off[CS];
    for (int k = tid; k < ncand; k += TP_THREADS) {
      int r = 0;
#pragma unroll
      for (int q = 1; q < CS; ++q) r += (k >= off[q]) ? 1 : 0;
      int base = 0;
#pragma unroll
      for (int q = 0; q < CS; ++q) base = (q == r) ? off[q] : base;
      const u64* rc = CS == 1 ? loc_comp : cluster.map_shared_rank(loc_comp, r);
      const uint32_t* rr = CS == 1 ? loc_rfix : cluster.map_shared_rank(loc_rfix, r);
      all_comp[k] = rc[k - base]; all_rfix[k] = rr[k - base];
    }
  }
  __syncthreads();

  // ---- exact cut: every CTA ranks its share of the candidates against all of them (8 threads per candidate, integer
  //      prefix masses); the one thread that finds the cut publishes it to every CTA of the cluster -----------------
  //      (Measured and dropped: one local radix level over the gathered candidates first -- a TP_NB-bin histogram of their
  //      composite keys, a block scan, the few candidates of the crossing bin compacted and ranked: its six block barriers
  //      at 1 024 threads cost what the quadratic ranking of ~500 candidates costs split over the CTAs of the row: Top-p
  //      24.8 against 24.4 us at config 2.)
  {
    const double trem = sh.trem;
    const int per = (ncand + CS - 1) / CS;
    const int i0 = rank * per, i1 = min(ncand, i0 + per);
    const int sub = tid & 7;
    for (int ib = i0; ib < i1; ib += TP_THREADS / 8) {
      const int i = ib + (tid >> 3);
      const bool valid = i < i1;
      const u64 ci = valid ? all_comp[i] : ~0ull;
      u64 P = 0;
      uint32_t rk = 0;
#pragma unroll 4
      for (int j = sub; j < ncand; j += 8) {                    // 8 consecutive candidates per warp load: conflict-free
        const bool ge = all_comp[j] >= ci;
        P += ge ? (u64)all_rfix[j] : 0ull;
        rk += ge ? 1u : 0u;
      }
#pragma unroll
      for (int o = 1; o < 8; o <<= 1) { P += __shfl_xor_sync(FULL, P, o); rk += __shfl_xor_sync(FULL, rk, o); }
      if (valid && sub == 0 && (double)P >= trem && (double)(P - all_rfix[i]) < trem) {
#pragma unroll
        for (int r = 0; r < CS; ++r) {
          TpSmall* ps = CS == 1 ? &sh : cluster.map_shared_rank(&sh, r);
          ps->cstar = ci; ps->ksel = sh.cnt_above + rk; ps->found = 1;
        }
      }
    }
  }
  TP_STAMP(7);
  csync();                                                    // S3: the cut is visible in every CTA
  TP_STAMP(8);
  if (!sh.found) {                                            // zero-weight candidates / rounding at the last ulp: take all of them
    if (tid == 0) {
      u64 mn = ~0ull;
      for (int j = 0; j < ncand; ++j) mn = min(mn, all_comp[j]);
      sh.cstar = mn; sh.ksel = sh.cnt_above + (uint32_t)ncand;
    }
    __syncthreads();
  }
  const u64 cstar = sh.cstar;
  const uint32_t total_sel = sh.ksel;

  // ---- pass 3: the candidates at or above the cut join the selection; bitmap words out (always), ascending index list
  //      (on request) ------------------------------------------------------------------------------------------------
  {
    const int nloc = min((int)sh.lcount, TP_CAND);
    for (int k = tid; k < nloc; k += TP_THREADS) {
      const u64 c = loc_comp[k];
      if (c >= cstar) {
        const int i = (int)(~(uint32_t)c) - lo;               // slice-local token index
        atomicOr(&selw[i >> 5], 1u << (i & 31));
      }
    }
    __syncthreads();
    for (int w = tid; w < nwords; w += TP_THREADS) bits_row[(lo >> 5) + w] = selw[w];
  }
  if (rank == 0 && tid == 0) sel_cnt[row] = (int32_t)total_sel;
  if (sel_idx) {
    __syncthreads();
    // exclusive scan of popc(selw) over the (<= TP_NB) words of the slice, TP_BPT words per thread
    uint32_t pc[TP_BPT], tsum = 0;
#pragma unroll
    for (int k = 0; k < TP_BPT; ++k) {
      const int w = TP_BPT * tid + k;
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
    for (int k = 0; k < TP_BPT; ++k) {
      const int w = TP_BPT * tid + k;
      if (w < nwords) woff[w] = run;
      run += pc[k];
    }
    if (tid == 0) sh.x_tot = tot;
    csync();                                                  // per-CTA totals visible
    uint32_t obase = 0;
#pragma unroll
    for (int r = 0; r < CS; ++r) if (r < rank) obase += peer(r)->x_tot;
    const unsigned lt = (1u << lane) - 1u;
    for (int w = warp; w < nwords; w += TP_WARPS) {
      const unsigned bal = selw[w];
      if ((bal >> lane) & 1u) sel_idx[rbase + obase + woff[w] + __popc(bal & lt)] = lo + w * 32 + lane;
    }
  }
  TP_STAMP(9);
  TP_STAMP(13);
  // keep shared memory alive until every peer has read it: after S3 only the index-list path reads a peer (x_tot)
  if (sel_idx) csync();
  TP_STAMP(14);
}

// order-preserving key of the row maximum, for caller-provided scores (rbq_topp_select); rowmax_key pre-zeroed
__global__ void rowmax_kernel(const float* __restrict__ scores, const int32_t* __restrict__ n_indexed, int Hq, int Lcap,
                              uint32_t* __restrict__ rowmax_key) {
  const int row = blockIdx.y, n = n_indexed[row / Hq];
  float mx = -INFINITY;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) mx = fmaxf(mx, scores[(size_t)row * Lcap + i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, o));
  if ((threadIdx.x & 31) == 0 && mx > -INFINITY) atomicMax(&rowmax_key[row], rbq_fkey(__fadd_rn(mx, 0.0f)));
}

template <int CS>
int launch_cs(rbq_ctx* ctx, const float* scores, uint32_t* rowmax_key, const int32_t* n_indexed, float p, uint32_t* bits,
              int wpr, int32_t* sel_idx, int32_t* sel_cnt, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int s_cap = ((((ctx->cfg.max_tokens + CS - 1) / CS) + 31) & ~31) + 32;
  const size_t smem = TP_OFF_SC + (size_t)s_cap * 4;
  auto kern = topp_kernel<CS>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_TOPP + CS, kern, RBQ_MAX_DYN_SMEM);
  dim3 grid(CS, rows);
  RBQ_CUDA_OK(ctx, rbq_launch_pdl(kern, grid, dim3(TP_THREADS), smem, s, scores, rowmax_key, n_indexed, ctx->cfg.n_q_heads,
                                  ctx->cfg.max_tokens, wpr, p, bits, sel_idx, sel_cnt));
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

}  // namespace

// Cluster size.  Few rows (<= one per SM): the largest of 8 / 4 / 2 / 1 CTAs per row that still gives every CTA an SM of its
// own (measured at config 2: 4 CTAs per row on 128 SMs make the step 6 us shorter than 8 per row with two CTAs on most
// SMs, although the kernel alone is 4 us longer -- its prologue overlaps the estimator's tail and it has half the exchange
// partners), as long as the slice fits in shared memory.  More rows than SMs: see below.
int rbq_topp_cluster_size(const rbq_ctx* ctx) {
  const long long rows = (long long)ctx->cfg.batch * ctx->cfg.n_q_heads;
  auto fits = [&](int c) {
    const long long s_cap = ((((ctx->cfg.max_tokens + c - 1) / c) + 31) & ~31) + 32;
    return TP_OFF_SC + (size_t)s_cap * 4 <= 227 * 1024 && s_cap <= 32 * TP_MAXW;
  };
  int cs = 8;
  if (rows <= ctx->sm_count) {
    while (cs > 1 && rows * cs > ctx->sm_count && fits(cs >> 1)) cs >>= 1;
    return cs;
  }
  // More rows than SMs: the smallest cluster whose slice fits.  Measured (512 rows, 16 K..64 K tokens): 277 / 260 /
  // 174 us at cluster size 8 / 4 / 2; (2 048 rows x 8 K): 298 / 162 / 89 us at 4 / 2 / 1 -- the fixed cost per CTA
  // (histogram set-up, cluster barriers) outweighs a second resident CTA per SM.
  while (cs > 1 && fits(cs >> 1)) cs >>= 1;
  return cs;
}

// rowmax_key == NULL: the maxima are computed here (rbq_topp_select on caller-provided scores).
int rbq_launch_topp(rbq_ctx* ctx, const float* scores, uint32_t* rowmax_key, const int32_t* n_indexed, float p,
                    uint32_t* sel_bits, int32_t* sel_idx, int32_t* sel_cnt, cudaStream_t s) {
  const int cs = rbq_topp_cluster_size(ctx);
  const int wpr = rbq_words_per_row(ctx);
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int s_cap = ((((ctx->cfg.max_tokens + cs - 1) / cs) + 31) & ~31) + 32;
  if (TP_OFF_SC + (size_t)s_cap * 4 > 227 * 1024 || s_cap > 32 * TP_MAXW)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select: max_tokens %d exceeds the cluster-resident limit", ctx->cfg.max_tokens);
  if (!rowmax_key) {
    uint32_t* rk = reinterpret_cast<uint32_t*>(static_cast<char*>(ctx->ws) + ctx->off_rowmax);
    RBQ_CUDA_OK(ctx, cudaMemsetAsync(rk, 0, (size_t)rows * sizeof(uint32_t), s));
    dim3 grid(max(1, min(32, (ctx->cfg.max_tokens + 4095) / 4096)), rows);
    rowmax_kernel<<<grid, 256, 0, s>>>(scores, n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, rk);
    RBQ_LAUNCH_OK(ctx);
    rowmax_key = rk;
  }
  switch (cs) {
    case 8: return launch_cs<8>(ctx, scores, rowmax_key, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    case 4: return launch_cs<4>(ctx, scores, rowmax_key, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    case 2: return launch_cs<2>(ctx, scores, rowmax_key, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
    default: return launch_cs<1>(ctx, scores, rowmax_key, n_indexed, p, sel_bits, wpr, sel_idx, sel_cnt, s);
  }
}

// the fp64 bin-edge tables of the Top-p kernel, once per context (the symbol is per device)
int rbq_topp_init(rbq_ctx* ctx) {
  double tab[TP_NC + 32];
  for (int k = 0; k < TP_NC; ++k) tab[k] = exp(-32.0 * (double)k / (double)TP_SCALE);
  for (int i = 0; i < 32; ++i) tab[TP_NC + i] = exp(-(double)i / (double)TP_SCALE);
  RBQ_CUDA_OK(ctx, cudaMemcpyToSymbol(g_tp_tab, tab, sizeof(tab)));
  return RBQ_OK;
}

// ---- rbq_topp_select_static: S6 on caller-provided scores with NO workspace and no allocation ----------------------------
// The scratch of the stage (the row-maximum keys and the per-row selection bitmaps the kernel always writes) lives in this
// file-scope device array: 2 MB that every GPU which loads the library holds until exit.  In host code the array's NAME is a
// host-side stand-in, not a device address: its device address comes from cudaGetSymbolAddress, once per device, with that
// device current.  Every call shares the array (contents of the last call stay; the keys are cleared per call): calls that
// overlap on the GPU race.
constexpr size_t TP_STATIC_WORDS = 512 * 1024;
static __device__ __align__(256) uint32_t g_tp_static_scratch[TP_STATIC_WORDS];
constexpr int TP_STATIC_MAX_DEVICES = 64;
static uint32_t* g_tp_static_addr[TP_STATIC_MAX_DEVICES];       // device address of the array on each device, 0 = not yet asked

int rbq_launch_topp_static(rbq_ctx* ctx, const float* scores, const int32_t* n_indexed, float p, int32_t* sel_idx,
                           int32_t* sel_cnt, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads, wpr = rbq_words_per_row(ctx);
  const size_t key_words = ((size_t)rows + 63) & ~size_t(63);   // bitmaps start 256-byte aligned
  const size_t need = key_words + (size_t)rows * wpr;
  if (need > TP_STATIC_WORDS)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED,
             "rbq_topp_select_static: batch*n_q_heads = %d rows x max_tokens %d need %zu bytes of scratch, the static array holds %zu "
             "(rows * (max_tokens / 32 + 1) must stay below ~%zu words); use rbq_topp_select with a workspace",
             rows, ctx->cfg.max_tokens, need * 4, TP_STATIC_WORDS * 4, TP_STATIC_WORDS);
  int dev = -1;
  RBQ_CUDA_OK(ctx, cudaGetDevice(&dev));
  if (dev < 0 || dev >= TP_STATIC_MAX_DEVICES) RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select_static: device ordinal %d", dev);
  if (!g_tp_static_addr[dev]) {                                   // set-up, once per device, that device current
    uint32_t* ptr = nullptr;
    RBQ_CUDA_OK(ctx, cudaGetSymbolAddress((void**)&ptr, g_tp_static_scratch));
    if (!ptr) RBQ_FAIL(ctx, RBQ_ERR_CUDA, "rbq_topp_select_static: no device address for the scratch array");
    g_tp_static_addr[dev] = ptr;
  }
  uint32_t* keys = g_tp_static_addr[dev];
  uint32_t* bits = keys + key_words;
  const int cs = rbq_topp_cluster_size(ctx);
  const int s_cap = ((((ctx->cfg.max_tokens + cs - 1) / cs) + 31) & ~31) + 32;
  if (TP_OFF_SC + (size_t)s_cap * 4 > 227 * 1024 || s_cap > 32 * TP_MAXW)
    RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "rbq_topp_select_static: max_tokens %d exceeds the cluster-resident limit", ctx->cfg.max_tokens);
  RBQ_CUDA_OK(ctx, cudaMemsetAsync(keys, 0, (size_t)rows * sizeof(uint32_t), s));   // the maxima are an atomicMax over zeroed keys
  dim3 grid(max(1, min(32, (ctx->cfg.max_tokens + 4095) / 4096)), rows);
  rowmax_kernel<<<grid, 256, 0, s>>>(scores, n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, keys);
  RBQ_LAUNCH_OK(ctx);
  switch (cs) {
    case 8: return launch_cs<8>(ctx, scores, keys, n_indexed, p, bits, wpr, sel_idx, sel_cnt, s);
    case 4: return launch_cs<4>(ctx, scores, keys, n_indexed, p, bits, wpr, sel_idx, sel_cnt, s);
    case 2: return launch_cs<2>(ctx, scores, keys, n_indexed, p, bits, wpr, sel_idx, sel_cnt, s);
    default: return launch_cs<1>(ctx, scores, keys, n_indexed, p, bits, wpr, sel_idx, sel_cnt, s);
  }
}

int rbq_probe_copy_topp(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, topp_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}
