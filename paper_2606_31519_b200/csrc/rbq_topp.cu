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
//   pass 1  : the slice is loaded by cp.async (whole slice in flight) and histogrammed: 2048 bins of width 1/64 in
//             u = m - score (monotone in C).  Per bin a (count, sum of r) pair, r = 2^(22 - (64u - j) log2(e)/64) in
//             2^-22 fixed point, so the bin mass is exp(-j/64) * sum(r): integer sums => order-independent, deterministic.
//             Only a 64-bin coarse summary (fp64) and then the 32 fine bins of the crossing coarse bin travel
//             through distributed shared memory (DSMEM is ~20 B/clk per SM).
//   pass 2  : ONE more pass over the resident slice classifies every token: bins above the crossing bin are selected (their
//             bitmap words are assembled right away), the tokens of the crossing bin (a few hundred at 128 K context) become
//             candidates; these are gathered from all CTAs in one DSMEM round; every CTA ranks its share of them against all
//             of them with integer prefix masses (8 threads per candidate) and the one thread that finds the cut C*
//             writes it into every CTA of the cluster.  If the crossing bin holds more than TP_CAND tokens (heavy ties),
//             it is first narrowed by cluster-wide 11-bit radix levels on C.
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

namespace {

constexpr int TP_THREADS = 512;
constexpr int TP_WARPS = TP_THREADS / 32;
constexpr int TP_NB = 4 * TP_THREADS;          // 2048 bins, 4 per thread in the scans
constexpr int TP_NC = 64;                      // coarse bins (32 fine bins each)
constexpr int TP_CAND = 1024;                  // candidates gathered per row
constexpr unsigned FULL = 0xffffffffu;
typedef unsigned long long u64;

struct TpSmall {
  u64 wt_u[TP_WARPS];
  uint32_t wt_c[TP_WARPS];
  u64 red_lo[TP_WARPS], red_hi[TP_WARPS];
  double tabA[TP_NC], tabB[32];                // exp(-k/2), exp(-i/64)
  // results broadcast inside the CTA
  double trem;            // mass still needed inside the candidate range, in units of 2^-22 * exp(-bx/64)
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
constexpr size_t TP_OFF_SC = TP_OFF_SELW + 2048 * sizeof(uint32_t);

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// fine bin j of u = m - s and the fixed-point residual weight r = exp(-(u - j/64)) * 2^22 = 2^(22 - (64u - j) log2(e)/64).
// The XU pipe (conversions, MUFU) is the scarce unit of the histogram pass, so floor() and both float <-> int conversions
// are done with the 2^23 magic-number add on the FMA pipe (round-down for the floor); only ex2 remains on the XU pipe.
// 2^-22 is the resolution of ex2.approx itself.
__device__ __forceinline__ void bin0(float m, float s, int& j, uint32_t& rfix) {
  const float t = __fmul_rn(__fsub_rn(m, s), 64.0f);          // >= 0
  const float jm = __fadd_rd(fminf(t, (float)(TP_NB - 1)), 8388608.0f);   // 2^23 + min(floor(t), TP_NB - 1), exact
  j = __float_as_int(jm) - 0x4B000000;
  const float f = __fsub_rn(t, __fsub_rn(jm, 8388608.0f));    // exact for j < TP_NB - 1; large in the overflow bin
  rfix = __float_as_uint(__fadd_rn(ex2_approx(fmaf(f, -0.022542110013890053f, 22.0f)), 8388608.0f)) - 0x4B000000u;
}
__device__ __forceinline__ u64 composite(float s, int t) {
  return ((u64)rbq_fkey(s) << 32) | (u64)(~(uint32_t)t);
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
// Pass-1 form of the histogram: three u32 arrays (mass bits 0..11, mass >> 12, count) updated by three independent
// reductions without return value -- no carry, so nothing waits for an atomic's result.  Sums stay below 2^32: at most
// 2^16 tokens per CTA with r < 2^23.  Folded into the (lo, count | hi) form after the pass.
__device__ __forceinline__ void hist_add3(uint32_t hist_sa, int j, u64 v, uint32_t c) {
  const uint32_t sa = hist_sa + 4u * (uint32_t)j;
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(sa), "r"((uint32_t)v & 0xFFFu) : "memory");
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(sa + 4u * TP_NB), "r"((uint32_t)(v >> 12)) : "memory");
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(sa + 8u * TP_NB), "r"(c) : "memory");
}
__device__ __forceinline__ void unpack_bin(uint2 v, uint32_t& cnt, u64& R) {
  cnt = v.y >> 12;
  R = ((u64)(v.y & 0xFFFu) << 32) | v.x;
}

// totals of this thread's 4 bins over the CS histograms of the cluster (cluster-wide radix levels only)
template <int CS>
__device__ __forceinline__ void gather_bins(cg::cluster_group& cluster, uint32_t* hist, int tid, uint32_t (&cnt)[4], u64 (&R)[4]) {
#pragma unroll
  for (int k = 0; k < 4; ++k) { cnt[k] = 0; R[k] = 0; }
#pragma unroll
  for (int r = 0; r < CS; ++r) {
    const uint32_t* rh = CS == 1 ? hist : cluster.map_shared_rank(hist, r);
    const uint4 a = reinterpret_cast<const uint4*>(rh)[tid], b = reinterpret_cast<const uint4*>(rh + TP_NB)[tid];
    uint32_t c; u64 v;
    unpack_bin(make_uint2(a.x, b.x), c, v); cnt[0] += c; R[0] += v;
    unpack_bin(make_uint2(a.y, b.y), c, v); cnt[1] += c; R[1] += v;
    unpack_bin(make_uint2(a.z, b.z), c, v); cnt[2] += c; R[2] += v;
    unpack_bin(make_uint2(a.w, b.w), c, v); cnt[3] += c; R[3] += v;
  }
}

// Integer block scan over TP_NB bins (4 per thread, ascending bin = descending C): finds the bin where the inclusive
// prefix of R first reaches sh.trem (clamped to the total), and updates sh.{trem, cnt_above, cntx, lo64, hi64}.
// `lo64`, `hi64`, `shift` describe the binning  bin = TP_NB-1 - ((C - lo64) >> shift).  Ends with a block barrier.
__device__ __forceinline__ void radix_scan(TpSmall& sh, const uint32_t (&cnt)[4], const u64 (&R)[4], u64 lo64, u64 hi64, int shift) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const u64 tsum = R[0] + R[1] + R[2] + R[3];
  const uint32_t csum = cnt[0] + cnt[1] + cnt[2] + cnt[3];
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
  u64 wp = 0, tot = 0;
  uint32_t wc = 0;
  for (int w = 0; w < TP_WARPS; ++w) { if (w < warp) { wp += sh.wt_u[w]; wc += sh.wt_c[w]; } tot += sh.wt_u[w]; }
  const double trem = fmin(trem_in, (double)tot);
  const u64 excl = wp + si - tsum, incl = wp + si;
  // exact integers: exactly one thread claims.  tot == 0 (every candidate weight underflows): first non-empty bin.
  const bool claim = tot > 0 ? ((double)excl < trem && (double)incl >= trem) : (wc + ci - csum == 0 && csum > 0);
  if (claim) {
    u64 c = excl;
    uint32_t cc = wc + ci - csum;
    int kx = -1;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (kx < 0) {
        if (tot > 0 ? ((double)(c + R[k]) >= trem) : (cnt[k] > 0)) kx = k;
        else { c += R[k]; cc += cnt[k]; }
      }
    }
    if (kx < 0) kx = 3;
    const int bsel = 4 * tid + kx;
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
__global__ void __cluster_dims__(CS, 1, 1) __launch_bounds__(TP_THREADS, 2)
topp_kernel(const float* __restrict__ scores, uint32_t* __restrict__ rowmax_key, const int32_t* __restrict__ n_indexed,
            int Hq, int Lcap, int wpr, float p_f, uint32_t* __restrict__ sel_bits, int32_t* __restrict__ sel_idx,
            int32_t* __restrict__ sel_cnt) {
  rbq_pdl_trigger();                                          // the wait for S5 comes after the shared-memory set-up
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
  for (int i = tid; i < 3 * TP_NB; i += TP_THREADS) hist[i] = 0u;   // third array: start of the candidate area, free until S1
  if (tid < TP_NC) sh.tabA[tid] = exp(-0.5 * (double)tid);
  else if (tid < TP_NC + 32) sh.tabB[tid - TP_NC] = exp(-0.015625 * (double)(tid - TP_NC));
  if (tid == 0) { sh.lcount = 0; sh.found = 0; }
  rbq_pdl_wait();                                             // scores and row maxima of S5
  TP_STAMP(1);
  const float m = __fadd_rn(rbq_fkey_inv(rowmax_key[row]), 0.0f);
  __syncthreads();
  {
    uint32_t of_c = 0;                                        // overflow bin kept in registers (can be half the row)
    u64 of_r = 0;
    const float4* src = reinterpret_cast<const float4*>(scores + rbase + lo);
    const int n4 = (len + 3) >> 2;                            // whole float4 groups (Lcap % 4 == 0: in bounds)
    // the whole slice in flight at once (16-byte cp.async, one latency round), then histogrammed from shared memory
    {
      const uint32_t sdst = (uint32_t)__cvta_generic_to_shared(sc);
      for (int i4 = tid; i4 < n4; i4 += TP_THREADS)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sdst + 16u * (uint32_t)i4), "l"(src + i4) : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
#pragma unroll 2
    for (int base = warp * 32; base < n4; base += TP_THREADS) {
      const int i4 = base + lane;
      float v[4] = {0.f, 0.f, 0.f, 0.f};
      if (i4 < n4) {                                            // each thread reads back exactly the groups it copied
        const float4 t4 = reinterpret_cast<const float4*>(sc)[i4];
        v[0] = __fadd_rn(t4.x, 0.0f); v[1] = __fadd_rn(t4.y, 0.0f); v[2] = __fadd_rn(t4.z, 0.0f); v[3] = __fadd_rn(t4.w, 0.0f);   // -0 -> +0
        reinterpret_cast<float4*>(sc)[i4] = make_float4(v[0], v[1], v[2], v[3]);
      }
      int j[4];
      uint32_t rf[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        j[k] = -1; rf[k] = 0;
        if (4 * i4 + k < len) bin0(m, v[k], j[k], rf[k]);
      }
      const int j0 = __shfl_sync(FULL, j[0], 0);
      if (__all_sync(FULL, j[0] == j0 && j[1] == j0 && j[2] == j0 && j[3] == j0)) {   // 128 tokens in one bin (ties)
        u64 t = (u64)rf[0] + rf[1] + rf[2] + rf[3];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(FULL, t, o);
        if (lane == 0) {
          if (j0 == TP_NB - 1) { of_c += 128; of_r += t; } else hist_add3(hist_sa, j0, t, 128u);
        }
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const bool of = j[k] == TP_NB - 1;
          of_c += of ? 1u : 0u;
          of_r += of ? (u64)rf[k] : 0ull;
          if (j[k] >= 0 && !of) hist_add3(hist_sa, j[k], (u64)rf[k], 1u);
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { of_c += __shfl_xor_sync(FULL, of_c, o); of_r += __shfl_xor_sync(FULL, of_r, o); }
    if (lane == 0 && of_c) hist_add3(hist_sa, TP_NB - 1, of_r, of_c);
  }
  __syncthreads();
  for (int b = tid; b < TP_NB; b += TP_THREADS) {               // fold into hist[b] = mass lo, hist[TP_NB + b] = count << 12 | mass hi
    const u64 mass = (u64)hist[b] + ((u64)hist[TP_NB + b] << 12);
    hist[b] = (uint32_t)mass;
    hist[TP_NB + b] = (hist[2 * TP_NB + b] << 12) | (uint32_t)(mass >> 32);
  }
  __syncthreads();
  // coarse summary of this CTA: 64 bins of 32 fine bins; thread t owns fine bins 4t..4t+3, 8 threads per coarse bin
  {
    double ms = 0.0;
    uint32_t cs = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint32_t c; u64 R;
      unpack_bin(make_uint2(hist[4 * tid + k], hist[TP_NB + 4 * tid + k]), c, R);
      ms += (double)R * sh.tabB[(4 * tid + k) & 31];
      cs += c;
    }
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) { ms += __shfl_xor_sync(FULL, ms, o); cs += __shfl_xor_sync(FULL, cs, o); }
    if ((tid & 7) == 0) { sh.xc_mass[tid >> 3] = ms * sh.tabA[tid >> 3]; sh.xc_cnt[tid >> 3] = cs; }
  }
  TP_STAMP(2);
  csync();                                                    // S1: histograms and coarse summaries complete
  TP_STAMP(3);
  if (rank == 0 && tid == 0) rowmax_key[row] = 0u;            // every CTA of the row has read its maximum: clear the key for the next step
  if (warp == 0) {
    // coarse crossing: lane l owns coarse bins 2l, 2l+1 (totals over the cluster in rank order), warp scan in fp64;
    // then the 32 fine bins of the crossing coarse bin, one per lane
    double m0 = 0.0, m1 = 0.0;
    uint32_t c0 = 0, c1 = 0;
#pragma unroll
    for (int r = 0; r < CS; ++r) {
      const TpSmall* ps = peer(r);
      m0 += ps->xc_mass[2 * lane]; m1 += ps->xc_mass[2 * lane + 1];
      c0 += ps->xc_cnt[2 * lane]; c1 += ps->xc_cnt[2 * lane + 1];
    }
    double si2 = m0 + m1;
    uint32_t ci2 = c0 + c1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double v = __shfl_up_sync(FULL, si2, o);
      const uint32_t cv = __shfl_up_sync(FULL, ci2, o);
      if (lane >= o) { si2 += v; ci2 += cv; }
    }
    const double Z = __shfl_sync(FULL, si2, 31);
    double T = (double)p_f * Z;
    const double ex2 = si2 - (m0 + m1);
    const uint32_t cex = ci2 - (c0 + c1);
    const bool x0 = c0 > 0 && ex2 + m0 >= T, x1 = c1 > 0 && (ex2 + m0) + m1 >= T;
    unsigned cb = __ballot_sync(FULL, x0 || x1);
    const unsigned ne = __ballot_sync(FULL, (c0 | c1) != 0);
    bool forced = false;
    if (cb == 0u) { cb = ne ? (1u << (31 - __clz(ne))) : 1u; forced = true; }   // rounding at the last ulp: last non-empty bin
    const int lsel = __ffs(cb) - 1;
    int kx = 0;
    double above = 0.0;
    uint32_t cab = 0;
    if (lane == lsel) {
      const bool second = forced ? (c1 > 0) : !x0;
      kx = 2 * lane + (second ? 1 : 0);
      above = second ? ex2 + m0 : ex2;
      cab = second ? cex + c0 : cex;
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
  const float u_lo = (float)bx * 0.015625f, u_hi = (bx == TP_NB - 1) ? INFINITY : (float)(bx + 1) * 0.015625f;
  bool use_range = false;

  // ---- heavy ties only: narrow the candidate range by cluster-wide 11-bit radix levels on C --------------
  if (cntx > TP_CAND) {
    u64 mn = ~0ull, mx = 0ull;
    for (int i = tid; i < len; i += TP_THREADS) {
      const float s = sc[i];
      const float u = __fsub_rn(m, s);
      if (u >= u_lo && u < u_hi) { const u64 c = composite(s, lo + i); mn = min(mn, c); mx = max(mx, c); }
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
      const int shift = max(0, (64 - __clzll((long long)range)) - 11);
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
            bin0(m, s, j_unused, rfix);
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
      uint32_t cnt[4];
      u64 R[4];
      gather_bins<CS>(cluster, hist, tid, cnt, R);
      radix_scan(sh, cnt, R, lo64, hi64, shift);
      csync();                                                // peers done reading this level's histogram
      lo64 = sh.lo64; hi64 = sh.hi64; cntx = sh.cntx;
      if (shift == 0) break;                                  // one C per bin: a single candidate is left
    }
  }

  // ---- pass 2: every token classified once: above the crossing bin -> its bit (8 lanes assemble one 32-token word);
  //      in the crossing bin (and, after a radix narrowing, inside the candidate range) -> local candidate list ----------
  {
    u64 lo64 = 0, hi64 = 0;
    if (use_range) { lo64 = sh.lo64; hi64 = sh.hi64; }
    const int n4r = nwords * 8;                               // float4 groups, rounded up to whole words
#pragma unroll 2
    for (int base = warp * 32; base < n4r; base += TP_THREADS) {
      const int i4 = base + lane;
      const float4 v4 = (i4 < n4r) ? reinterpret_cast<const float4*>(sc)[i4] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float v[4] = {v4.x, v4.y, v4.z, v4.w};
      uint32_t nib = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int i = 4 * i4 + k;
        const float u = __fsub_rn(m, v[k]);
        bool sel = (i < len) && (u < u_lo);
        if (i < len && u >= u_lo && u < u_hi) {
          const u64 c = composite(v[k], lo + i);
          if (!use_range || (c >= lo64 && c <= hi64)) {
            int j_unused;
            uint32_t rfix;
            bin0(m, v[k], j_unused, rfix);
            const uint32_t slot = atomicAdd(&sh.lcount, 1u);
            if (slot < TP_CAND) { loc_comp[slot] = c; loc_rfix[slot] = rfix; }
          } else if (c > hi64) {
            sel = true;                                       // narrowed range: above it = selected for sure
          }
        }
        nib |= sel ? (1u << k) : 0u;
      }
      uint32_t word = nib << (4 * (lane & 7));
      word |= __shfl_xor_sync(FULL, word, 1);
      word |= __shfl_xor_sync(FULL, word, 2);
      word |= __shfl_xor_sync(FULL, word, 4);
      if ((lane & 7) == 0 && i4 < n4r) selw[i4 >> 3] = word;
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
  csync();                                                    // keep shared memory alive until every peer has read it
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
    return TP_OFF_SC + (size_t)s_cap * 4 <= 227 * 1024 && s_cap <= 32 * TP_NB;
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
  if (TP_OFF_SC + (size_t)s_cap * 4 > 227 * 1024 || s_cap > 32 * TP_NB)
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

int rbq_probe_copy_topp(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, topp_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}
