// rbq_attention.cu -- S7: exact attention over the gathered selected tokens and the pending window
// (Alg.2 lines 14-15, L188-190; L215 "K_local ... participate in the hybrid attention";
// renormalised over the attended set, R7).
//
// The stage is an HBM-bound gather: 2*D*sizeof(T) bytes per attended (token, KV head).  The G query
// heads of a KV group select different but overlapping sets, so the least the method must move is the
// UNION of the group's sets -- that is what this path fetches, once:
//   attn_plan_kernel   per KV group: OR of the G per-head selection bitmaps (written by S6) ->
//                      compact ascending union list, entry = token | (head mask << 28), + its length.
//   attn_gather_kernel persistent, one CTA per SM.  The concatenated union lists (+ pending windows) of
//                      all groups are cut into equal contiguous ranges, one per CTA; inside a CTA each
//                      warp runs a private 3-stage cp.async pipeline of 16-row K/V tiles (swizzled
//                      shared memory, 128 KB in flight per SM) and contracts them on the tensor pipe:
//                      S[head, token] = Q K^T and O += P V with mma.sync.m16n8k16.bf16 (heads on M, so
//                      softmax statistics stay inside a quad, as in FlashAttention-2), head masks applied
//                      to S.  The dot products are tiny (4*D FLOP per row and head); the tensor pipe is used
//                      because it leaves the issue slots to the address generation of the gather.
//                      The last CTA to finish a group (arrival counter) merges the group's (m, l, o) partials
//                      into out / lse, so no merge launch sits on the critical path.
// fp32 K/V or q (parity config 0) take the FP32-pipe kernel attn_simt_kernel over the same union lists.
#include "rbq_common.cuh"

RBQ_PROBE_DECL(gather_probe);
RBQ_PROBE_DECL(plan_probe);
#ifdef RBQ_PROBE
#define PL_STAMP(slot)                                                                                           \
  do {                                                                                                           \
    const unsigned cta_ = blockIdx.y * gridDim.x + blockIdx.x;                                                    \
    if (threadIdx.x == 0 && cta_ < RBQ_PROBE_CTAS) {                                                              \
      plan_probe[cta_ * RBQ_PROBE_SLOTS + (slot)] = (unsigned long long)clock64();                                \
      if ((slot) == 0) { unsigned long long gt_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_)); plan_probe[cta_ * RBQ_PROBE_SLOTS + 15] = gt_; } \
    }                                                                                                            \
  } while (0)
#else
#define PL_STAMP(slot) do {} while (0)
#endif

namespace {

// ---- bitmaps from caller-provided index lists (stand-alone rbq_sparse_attention) --------------------------------
__global__ void bits_from_lists_kernel(const int32_t* __restrict__ sel_idx, const int32_t* __restrict__ sel_cnt,
                                       const int32_t* __restrict__ n_indexed, int Hq, int Lcap, int wpr,
                                       uint32_t* __restrict__ bits) {
  const int row = blockIdx.y, b = row / Hq;
  const int cnt = min(sel_cnt[row], Lcap), n = n_indexed[b];
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += gridDim.x * blockDim.x) {
    const int t = sel_idx[(size_t)row * Lcap + i];
    if (t >= 0 && t < n) atomicOr(&bits[(size_t)row * wpr + (t >> 5)], 1u << (t & 31));
  }
}

// ---- plan: union list per KV group ---------------------------------------------------------------------------------
constexpr int PL_THREADS = 1024;
constexpr int PL_MAX_SPLIT = 16;

// grid = (PL_SPLIT, B*Hkv); PL_SPLIT = the largest of 16, 8, 4, 2, 1 that keeps the grid within one wave (one CTA per
// SM: with two per SM assumed, configs 3 and 4 ran 256 CTAs in two waves).  Every CTA of a group recomputes the prefix over
// the 128-token blocks (one block per thread: 4 words x G heads), then its warps expand the blocks with
// blk % PL_SPLIT == blockIdx.x cooperatively (lane = token bit of a word, position by popcount prefix).
// Measured and dropped (config 4, in-kernel stamps: 5.5 K cycles of loads + scan, 12 K cycles of expansion): one word per
// thread walking the set bits, with direct stores (32 scattered 4-byte transactions per instruction) or staged through
// 32 KB of shared memory and written out coalesced with entry-balanced contiguous shares -- the expansion stayed at
// 11-13 K cycles (37 % of the union's bits are set there: ~25 issue slots per entry either way) and the step got slower
// (config 4: 271 -> 283-288 us).
template <int PL_SPLIT>
__global__ void __launch_bounds__(PL_THREADS)
attn_plan_kernel(const uint32_t* __restrict__ bits, const int32_t* __restrict__ n_indexed, const int32_t* __restrict__ n_total,
                 int Hq, int Hkv, int Lcap, int wpr, uint32_t* __restrict__ ulist, int32_t* __restrict__ ucount,
                 int32_t* __restrict__ gdone) {
  __shared__ uint32_t s_warp[PL_THREADS / 32];
  __shared__ uint32_t s_pre[PL_THREADS], s_cntb[PL_THREADS];
  __shared__ uint32_t s_base;
  rbq_pdl_trigger();
  PL_STAMP(0);
  const int gi = blockIdx.y, b = gi / Hkv, g = gi % Hkv, G = Hq / Hkv;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // n_indexed is an input of the step (committed before S3, which starts only when the kernel in front of it has
  // completed): loaded before the wait, one dependent round trip less behind it
  const int nidx = max(0, n_indexed[b]);
  rbq_pdl_wait();                                             // selection bitmaps of S6
  PL_STAMP(1);
  const int nw = (nidx + 31) >> 5, nblk = (nw + 3) >> 2;
  const uint32_t* rows0 = bits + ((size_t)b * Hq + (size_t)g * G) * wpr;
  uint32_t* __restrict__ out = ulist + (size_t)gi * Lcap;
  if (tid == 0) s_base = 0;
  __syncthreads();
  for (int blk0 = 0; blk0 < nblk; blk0 += PL_THREADS) {
    const int blk = blk0 + tid;
    uint32_t uw[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int h = 0; h < RBQ_MAX_G; ++h) {
      uint4 v = make_uint4(0u, 0u, 0u, 0u);
      if (h < G && blk < nblk) v = *reinterpret_cast<const uint4*>(rows0 + (size_t)h * wpr + 4 * blk);
      uw[0] |= v.x; uw[1] |= v.y; uw[2] |= v.z; uw[3] |= v.w;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) if (4 * blk + k >= nw) uw[k] = 0u;   // words beyond the indexed prefix were never written
    const uint32_t c = __popc(uw[0]) + __popc(uw[1]) + __popc(uw[2]) + __popc(uw[3]);
    uint32_t si = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += v;
    }
    if (lane == 31) s_warp[warp] = si;
    __syncthreads();
    uint32_t wp = 0, tot = 0;
    for (int w = 0; w < PL_THREADS / 32; ++w) { if (w < warp) wp += s_warp[w]; tot += s_warp[w]; }
    s_pre[tid] = s_base + wp + si - c;
    s_cntb[tid] = c;
    __syncthreads();
    PL_STAMP(2);
    // this warp's blocks: lb = blockIdx.x + PL_SPLIT * (warp + 32 i), i < PL_BPW.  Lane l < 16 prefetches word (l & 3) of head
    // (l >> 2) of each block first (one round of independent loads), then the words are broadcast by shuffles.
    const unsigned lt = (1u << lane) - 1u;
    constexpr int PL_BPW = PL_THREADS / (PL_SPLIT * (PL_THREADS / 32));          // blocks per warp and iteration
    uint32_t pre[PL_BPW];
#pragma unroll
    for (int i = 0; i < PL_BPW; ++i) {
      const int lb = (int)blockIdx.x + PL_SPLIT * (warp + (PL_THREADS / 32) * i);
      const int wi = 4 * (blk0 + lb) + (lane & 3), h = lane >> 2;
      pre[i] = (lane < 16 && h < G && blk0 + lb < nblk && wi < nw && s_cntb[lb] != 0) ? rows0[(size_t)h * wpr + wi] : 0u;
    }
#pragma unroll
    for (int i = 0; i < PL_BPW; ++i) {
      const int lb = (int)blockIdx.x + PL_SPLIT * (warp + (PL_THREADS / 32) * i);
      const int bk = blk0 + lb;
      if (bk >= nblk || s_cntb[lb] == 0) continue;              // warp-uniform
      uint32_t pos = s_pre[lb];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        uint32_t u = 0, mask = 0;
#pragma unroll
        for (int h = 0; h < RBQ_MAX_G; ++h) {
          const uint32_t hwv = __shfl_sync(0xffffffffu, pre[i], 4 * h + k);
          u |= hwv;
          mask |= ((hwv >> lane) & 1u) << h;
        }
        if ((u >> lane) & 1u) out[pos + __popc(u & lt)] = (uint32_t)((4 * bk + k) * 32 + lane) | (mask << 28);
        pos += __popc(u);
      }
    }
    PL_STAMP(3);
    __syncthreads();
    if (tid == 0) s_base += tot;
    __syncthreads();
  }
  PL_STAMP(4);
  if (blockIdx.x == 0 && tid == 0) { ucount[gi] = (int32_t)s_base; gdone[gi] = 0; }
}

// ---- shared by the gather kernels: exclusive prefix of attended rows per group ----------------------------------
constexpr int AT_MAX_GROUPS = 1024;

// s_start[gi] = sum over groups < gi of (ucount + pending); s_start[ngroups] = total.  Every CTA computes the same table.
// s_ucnt / s_nidx (or NULL): per-group copies of ucount and the sequence's indexed count, so that the caller needs no
// second global round trip for them.
__device__ void build_group_table(const int32_t* __restrict__ ucount, const int32_t* __restrict__ n_indexed,
                                  const int32_t* __restrict__ n_total, int ngroups, int Hkv, int* s_start, int* s_warp,
                                  int nthreads, int* s_ucnt = nullptr, int* s_nidx = nullptr) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
  const int per = (ngroups + nthreads - 1) / nthreads;
  const int g0 = tid * per;
  int local = 0;
  for (int gi = g0; gi < min(ngroups, g0 + per); ++gi) {
    const int b = gi / Hkv;
    const int uc = ucount[gi], ni = max(0, n_indexed[b]);
    if (s_ucnt) { s_ucnt[gi] = uc; s_nidx[gi] = ni; }
    local += uc + max(0, n_total[b] - ni);
  }
  int incl = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int woff = 0, total = 0;
  for (int w = 0; w < nwarps; ++w) { if (w < warp) woff += s_warp[w]; total += s_warp[w]; }
  int run = woff + incl - local;
  for (int gi = g0; gi < min(ngroups, g0 + per); ++gi) {
    const int b = gi / Hkv;
    s_start[gi] = run;
    run += ucount[gi] + max(0, n_total[b] - max(0, n_indexed[b]));
  }
  if (tid == 0) s_start[ngroups] = total;
  __syncthreads();
}

// Work partition of the gather: contiguous ranges of the concatenated attended rows, one per CTA, of equal COST: starting a
// KV group inside a CTA's range costs a second prologue and merge, so every group start (but the first) counts as GA_PEN
// virtual rows: the ranges are equal in that virtual space and mapped back to rows -- a CTA that contains a group start
// gets that many fewer rows, and a boundary falling into a gap snaps to the group's first row.  Measured at config 2 (stage
// events): 56.3 / 55.6 / 57.5 us at GA_PEN = 0 / 320 / 640 -- a small effect: the kernel streams at the copy peak
// (235.5 MB in 37 us once the first tiles are requested, profiles/r02_ncu.md).  Snapping ALL boundaries to group
// boundaries was measured too: worse, a group worth 1.4 CTAs rounds to one.
constexpr int GA_PEN = 320;
// virtual coordinate v in [0, total + GA_PEN * (ngroups - 1)]  ->  row in [0, total]; monotone, every CTA computes the same
__device__ __forceinline__ long long ga_row_of(const int* s_start, int ngroups, long long v) {
  int lo = 0, hi = ngroups - 1;                               // last group whose virtual start s_start[gi] + GA_PEN * gi is <= v
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if ((long long)s_start[mid] + (long long)GA_PEN * mid <= v) lo = mid; else hi = mid - 1;
  }
  const long long off = v - ((long long)s_start[lo] + (long long)GA_PEN * lo) - (lo > 0 ? GA_PEN : 0);   // rows into the group
  const long long rows = (long long)s_start[lo + 1] - s_start[lo];
  return s_start[lo] + min(max(off, 0ll), rows);
}
// first row of CTA c's range: floor(vtot * c / nc) in 32-bit integer arithmetic (vtot = q0 nc + r0: q0 c + floor(r0 c / nc),
// r0 c < nc^2); identical in every CTA.  (fp64 here cost ~1.5 K cycles of dependent DFMAs on the critical path of every
// CTA, a 64-bit division about as much.)
__device__ __forceinline__ long long cta_begin(const int* s_start, int ngroups, long long total, int c, int nc) {
  if (c >= nc) return total;
  const unsigned vtot = (unsigned)(total + (long long)GA_PEN * (ngroups - 1));       // < 2^31 + 320 * 1024
  const unsigned q0 = vtot / (unsigned)nc, r0 = vtot - q0 * (unsigned)nc;
  return ga_row_of(s_start, ngroups, (long long)q0 * c + (long long)((r0 * (unsigned)c) / (unsigned)nc));
}

// ---- tensor-pipe gather attention (bf16 K/V and q) ----------------------------------------------------------------------
#ifndef RBQ_GA_WARPS
#define RBQ_GA_WARPS 8
#endif
#ifndef RBQ_GA_STAGES
#define RBQ_GA_STAGES 3
#endif
constexpr int GA_WARPS = RBQ_GA_WARPS;
constexpr int GA_THREADS = GA_WARPS * 32;
constexpr int GA_STAGES = RBQ_GA_STAGES;
constexpr int GA_TILE = 16;                                   // rows per warp tile
// per head_dim D (template parameter, 64 or 128; D = 256 takes the FP32-pipe kernel below):
template <int D> struct GaCfg {
  static constexpr int ROW_BYTES = D * 2;                     // one bf16 K or V row
  static constexpr int CPR = D / 8;                           // 16-byte chunks per row
  static constexpr int TILE_BYTES = GA_TILE * ROW_BYTES;      // 4 KB per operand at D = 128
  static constexpr int STAGE_BYTES = 2 * TILE_BYTES;          // K + V
  static constexpr int SMEM = GA_WARPS * GA_STAGES * STAGE_BYTES;   // 192 KB at D = 128
  static constexpr int PART = D + 4;                          // floats per (partial, head): o[D], m (base-2 units), l, pad (16-byte rows)
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&v);
}

// grid = number of SMs (persistent), GA_THREADS threads, GaCfg<D>::SMEM dynamic shared memory.
// part: [gridDim.x + ngroups][G][GA_PART]; the partial of (CTA c, group gi) lives in slot c + gi.
template <int D>
__global__ void __launch_bounds__(GA_THREADS, 1)
attn_gather_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ K, const __nv_bfloat16* __restrict__ V,
                   long long sb, long long sh, long long st, const uint32_t* __restrict__ ulist,
                   const int32_t* __restrict__ ucount, const int32_t* __restrict__ n_indexed,
                   const int32_t* __restrict__ n_total, int ngroups, int Hq, int Hkv, int Lcap, float scale_log2,
                   float* __restrict__ part, int32_t* __restrict__ gdone, void* __restrict__ out, int out_bf16,
                   float* __restrict__ lse) {
  using C = GaCfg<D>;
  constexpr int GA_TILE_BYTES = C::TILE_BYTES, GA_STAGE_BYTES = C::STAGE_BYTES, GA_PART = C::PART, RB = C::ROW_BYTES, CPR = C::CPR;
  constexpr int LSH = (D == 64) ? 3 : 4;                       // log2(CPR)
  extern __shared__ __align__(128) unsigned char ga_smem[];
  __shared__ int s_start[AT_MAX_GROUPS + 1], s_ucnt[AT_MAX_GROUPS], s_nidx[AT_MAX_GROUPS];
  __shared__ int s_warp[GA_WARPS];
  __shared__ int s_last, s_clo, s_chi;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g4 = lane >> 2, t4 = lane & 3;                    // MMA fragment coordinates
  const int G = Hq / Hkv;
  if (tid == 0) RBQ_STAMP(gather_probe, 0);
  rbq_pdl_wait();                                             // union lists of the plan kernel
  if (tid == 0) RBQ_STAMP(gather_probe, 1);

  build_group_table(ucount, n_indexed, n_total, ngroups, Hkv, s_start, s_warp, GA_THREADS, s_ucnt, s_nidx);
  if (tid == 0) RBQ_STAMP(gather_probe, 2);
  const long long total = s_start[ngroups];
  if (blockIdx.x == 0) {                                      // groups with nothing to attend: out = 0, lse = -inf
    for (int gq = 0; gq < ngroups; ++gq) {
      if (s_start[gq + 1] != s_start[gq]) continue;
      for (int hd = tid; hd < G * D; hd += GA_THREADS) {
        const size_t orow = (size_t)(gq / Hkv) * Hq + (size_t)(gq % Hkv) * G + hd / D;
        if (out_bf16) reinterpret_cast<__nv_bfloat16*>(out)[orow * D + hd % D] = __float2bfloat16_rn(0.0f);
        else reinterpret_cast<float*>(out)[orow * D + hd % D] = 0.0f;
        if (lse && hd % D == 0) lse[orow] = -INFINITY;
      }
    }
  }
  const long long r0 = cta_begin(s_start, ngroups, total, blockIdx.x, gridDim.x), r1 = cta_begin(s_start, ngroups, total, blockIdx.x + 1, gridDim.x);
  if (r0 >= r1) return;
  // first group with s_start[gi + 1] > r0
  int gi = 0;
  {
    int lo = 0, hi = ngroups - 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if ((long long)s_start[mid + 1] > r0) hi = mid; else lo = mid + 1;
    }
    gi = lo;
  }
  if (tid == 0) RBQ_STAMP(gather_probe, 9);
  unsigned char* my_smem = ga_smem + (size_t)warp * GA_STAGES * GA_STAGE_BYTES;
  const uint32_t my_base = smem_u32(my_smem);

  for (; gi < ngroups && (long long)s_start[gi] < r1; ++gi) {
    const long long ga = s_start[gi], gb = s_start[gi + 1];
    const int a = (int)(max(r0, ga) - ga), e = (int)(min(r1, gb) - ga);   // group-local rank range of this CTA
    if (a >= e) continue;
    const int b = gi / Hkv, g = gi % Hkv;
    const int usel = s_ucnt[gi], nidx = s_nidx[gi];
    const __nv_bfloat16* Kb = K + (long long)b * sb + (long long)g * sh;
    const __nv_bfloat16* Vb = V + (long long)b * sb + (long long)g * sh;
    const uint32_t* ul = ulist + (size_t)gi * Lcap;

    if (tid == 0) RBQ_STAMP(gather_probe, 12);
    // A operand: Q rows of the group's heads (rows >= G are zero)
    uint32_t qa[D / 16][2];
    {
      const uint32_t* qp = reinterpret_cast<const uint32_t*>(q + ((size_t)b * Hq + (size_t)g * G + min(g4, G - 1)) * D);
#pragma unroll
      for (int ks = 0; ks < D / 16; ++ks) {
        qa[ks][0] = (g4 < G) ? qp[8 * ks + t4] : 0u;
        qa[ks][1] = (g4 < G) ? qp[8 * ks + 4 + t4] : 0u;
      }
    }
    if (tid == 0) RBQ_STAMP(gather_probe, 10);
    float m_run = -INFINITY, l_run = 0.0f;
    float o[D / 8][4];
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt) { o[nt][0] = 0.0f; o[nt][1] = 0.0f; o[nt][2] = 0.0f; o[nt][3] = 0.0f; }

    const int ntiles = (e - a + GA_TILE - 1) / GA_TILE;
    const int my_tiles = (ntiles > warp) ? (ntiles - warp + GA_WARPS - 1) / GA_WARPS : 0;

    // entry of row `lane` (lanes 0..15) of tile i of this warp: token | mask << 28 (mask 0 = padding row)
    auto tile_entry = [&](int i) -> uint32_t {
      const int r = a + (warp + i * GA_WARPS) * GA_TILE + lane;
      uint32_t ent = 0u;
      if (lane < GA_TILE && r < e) ent = (r < usel) ? ul[r] : ((uint32_t)(nidx + (r - usel)) | (0xFu << 28));
      return ent;
    };
    auto issue = [&](int i, uint32_t ent) {
      const uint32_t sbase = my_base + (uint32_t)((i % GA_STAGES) * GA_STAGE_BYTES);
#pragma unroll
      for (int k = 0; k < GA_TILE * CPR / 32; ++k) {           // 32 lanes cover 32 / CPR rows per step
        const int row = (32 / CPR) * k + (lane >> LSH), ch = lane & (CPR - 1);
        const uint32_t re = __shfl_sync(0xffffffffu, ent, row);
        const long long off = (long long)(re & 0x0FFFFFFFu) * st + ch * 8;
        const uint32_t d = sbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4));
        cp_async16(d, Kb + off);
        cp_async16(d + GA_TILE_BYTES, Vb + off);
      }
    };
    // entries of the tiles in flight (ring) and of the next tile to issue, loaded one iteration ahead so that the
    // index load never sits between a freed stage and its refill
    uint32_t ent_ring[GA_STAGES - 1], ent_pend;
#pragma unroll
    for (int s = 0; s < GA_STAGES - 1; ++s) ent_ring[s] = (s < my_tiles) ? tile_entry(s) : 0u;
    ent_pend = (GA_STAGES - 1 < my_tiles) ? tile_entry(GA_STAGES - 1) : 0u;
    if (tid == 0) RBQ_STAMP(gather_probe, 11);
#pragma unroll
    for (int s = 0; s < GA_STAGES - 1; ++s) {
      if (s < my_tiles) issue(s, ent_ring[s]);
      cp_async_commit();
    }
    if (tid == 0) RBQ_STAMP(gather_probe, 3);
    for (int i = 0; i < my_tiles; ++i) {
      const uint32_t ent = ent_ring[0];
      const int nx = i + GA_STAGES - 1;
      if (nx < my_tiles) issue(nx, ent_pend);
#pragma unroll
      for (int s = 0; s + 1 < GA_STAGES - 1; ++s) ent_ring[s] = ent_ring[s + 1];
      ent_ring[GA_STAGES - 2] = ent_pend;
      ent_pend = (nx + 1 < my_tiles) ? tile_entry(nx + 1) : 0u;
      cp_async_commit();
      cp_async_wait<GA_STAGES - 1>();
      __syncwarp();
      if (tid == 0 && i == 0) RBQ_STAMP(gather_probe, 4);
      const uint32_t kbase = my_base + (uint32_t)((i % GA_STAGES) * GA_STAGE_BYTES), vbase = kbase + GA_TILE_BYTES;

      // S = Q K^T : two n-tiles of 8 tokens
      float s[2][4];
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        s[nt][0] = 0.0f; s[nt][1] = 0.0f; s[nt][2] = 0.0f; s[nt][3] = 0.0f;
        const int row = nt * 8 + (lane & 7);
#pragma unroll
        for (int j = 0; j < D / 32; ++j) {
          uint32_t bf[4];
          const int ch = 4 * j + (lane >> 3);
          ldsm_x4(bf, kbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4)));
          mma_bf16(s[nt], qa[2 * j][0], 0u, qa[2 * j][1], 0u, bf[0], bf[1]);
          mma_bf16(s[nt], qa[2 * j + 1][0], 0u, qa[2 * j + 1][1], 0u, bf[2], bf[3]);
        }
      }
      // head masks, online softmax (row = head g4; this lane: tokens nt*8 + 2*t4, +1)
      float tmax = -INFINITY;
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const uint32_t e0 = __shfl_sync(0xffffffffu, ent, nt * 8 + 2 * t4);
        const uint32_t e1 = __shfl_sync(0xffffffffu, ent, nt * 8 + 2 * t4 + 1);
        const bool ok0 = (e0 >> (28 + (g4 & 3))) & 1u, ok1 = (e1 >> (28 + (g4 & 3))) & 1u;
        s[nt][0] = (ok0 && g4 < G) ? s[nt][0] * scale_log2 : -INFINITY;
        s[nt][1] = (ok1 && g4 < G) ? s[nt][1] * scale_log2 : -INFINITY;
        tmax = fmaxf(tmax, fmaxf(s[nt][0], s[nt][1]));
      }
      tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
      tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
      const float m_new = fmaxf(m_run, tmax);
      const float m_use = (m_new == -INFINITY) ? 0.0f : m_new;
      const float resc = exp2f(m_run - m_use);                 // m_run = -inf -> 0
      m_run = m_new;
      const float p00 = exp2f(s[0][0] - m_use), p01 = exp2f(s[0][1] - m_use);
      const float p10 = exp2f(s[1][0] - m_use), p11 = exp2f(s[1][1] - m_use);
      l_run = l_run * resc + ((p00 + p01) + (p10 + p11));
      // P as bf16 hi + lo parts (two MMAs per V tile): keeps ~16 mantissa bits of the probabilities
      const uint32_t pa0 = pack_bf16(p00, p01), pa2 = pack_bf16(p10, p11);
      const uint32_t pb0 = pack_bf16(p00 - rbq_bf16lo(pa0), p01 - rbq_bf16hi(pa0));
      const uint32_t pb2 = pack_bf16(p10 - rbq_bf16lo(pa2), p11 - rbq_bf16hi(pa2));
      // O = O * resc + P V
#pragma unroll
      for (int c2 = 0; c2 < D / 16; ++c2) {
        uint32_t bf[4];
        const int row = (lane & 7) + ((lane >> 3) & 1) * 8, ch = 2 * c2 + (lane >> 4);
        ldsm_x4_t(bf, vbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4)));
        o[2 * c2][0] *= resc; o[2 * c2][1] *= resc;
        o[2 * c2 + 1][0] *= resc; o[2 * c2 + 1][1] *= resc;
        mma_bf16(o[2 * c2], pa0, 0u, pa2, 0u, bf[0], bf[1]);
        mma_bf16(o[2 * c2 + 1], pa0, 0u, pa2, 0u, bf[2], bf[3]);
        mma_bf16(o[2 * c2], pb0, 0u, pb2, 0u, bf[0], bf[1]);
        mma_bf16(o[2 * c2 + 1], pb0, 0u, pb2, 0u, bf[2], bf[3]);
      }
      __syncwarp();                                            // tile consumed before its stage is refilled
    }
    cp_async_wait<0>();
    rbq_pdl_trigger();                                        // dependents (the next step's S3) may become resident under the merge phase
    if (tid == 0) RBQ_STAMP(gather_probe, 5);
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);

    // merge the warps of the CTA (staging area aliases the drained pipeline buffers)
    __syncthreads();
    float* stg = reinterpret_cast<float*>(ga_smem);            // [GA_WARPS][G][GA_PART]
    if (g4 < G) {
      float* dst = stg + ((size_t)warp * G + g4) * GA_PART;
#pragma unroll
      for (int nt = 0; nt < D / 8; ++nt) { dst[8 * nt + 2 * t4] = o[nt][0]; dst[8 * nt + 2 * t4 + 1] = o[nt][1]; }
      if (t4 == 0) { dst[D] = m_run; dst[D + 1] = l_run; }
    }
    __syncthreads();
    float* pdst = part + (size_t)(blockIdx.x + gi) * G * GA_PART;
    for (int idx = tid; idx < G * D; idx += GA_THREADS) {
      const int h = idx / D, d = idx % D;
      float mm = -INFINITY;
#pragma unroll
      for (int w = 0; w < GA_WARPS; ++w) mm = fmaxf(mm, stg[((size_t)w * G + h) * GA_PART + D]);
      float oo = 0.0f, ll = 0.0f;
#pragma unroll
      for (int w = 0; w < GA_WARPS; ++w) {
        const float* sp = stg + ((size_t)w * G + h) * GA_PART;
        const float f = (sp[D] == -INFINITY) ? 0.0f : exp2f(sp[D] - mm);
        oo = fmaf(f, sp[d], oo);
        ll = fmaf(f, sp[D + 1], ll);
      }
      pdst[(size_t)h * GA_PART + d] = oo;
      if (d == 0) { pdst[(size_t)h * GA_PART + D] = mm; pdst[(size_t)h * GA_PART + D + 1] = ll; }
    }
    // ---- arrival: the last CTA that finishes a group merges the group's partials into out / lse -------------------------
    if (tid == 0) RBQ_STAMP(gather_probe, 6);
    __threadfence();
    const int nc = (int)gridDim.x;
    const bool touches = tid < nc && max(cta_begin(s_start, ngroups, total, tid, nc), ga) < min(cta_begin(s_start, ngroups, total, tid + 1, nc), gb);
    if (tid == 0) { s_clo = nc; s_chi = -1; }
    const int expected = __syncthreads_count(touches);         // also: staging area free, partial stores fenced
    if (touches) { atomicMin(&s_clo, tid); atomicMax(&s_chi, tid); }
    if (tid == 0) s_last = (atomicAdd(&gdone[gi], 1) == expected - 1);
    __syncthreads();
    if (tid == 0) RBQ_STAMP(gather_probe, 7);
    if (s_last) {
      __threadfence();
      float* s_f = stg;                                        // [G][GA_THREADS]: factor 2^(m - max) of slot c
      constexpr int TPH = D / 4, ITEMS = RBQ_MAX_G * TPH;     // threads per head (4 dims each), (head, dim group) items
      constexpr int NH = GA_THREADS / ITEMS;                   // slot subsets worked on in parallel (2 at D = 128, 4 at D = 64)
      float4* s_o = reinterpret_cast<float4*>(stg + 2 * RBQ_MAX_G * GA_THREADS);   // [NH - 1][ITEMS] partial sums of subsets 1 ..
      const int clo = s_clo, chi = s_chi;
      // thread tid owns slot tid: per-head maximum and normaliser by block reductions (warp shuffles + one shared round)
      float* s_red = stg + 2 * RBQ_MAX_G * GA_THREADS + 4 * (NH > 1 ? (NH - 1) * ITEMS : 1);   // [2][RBQ_MAX_G][GA_WARPS]
      float pm[RBQ_MAX_G], pl[RBQ_MAX_G];
#pragma unroll
      for (int h = 0; h < RBQ_MAX_G; ++h) {
        pm[h] = -INFINITY; pl[h] = 0.0f;
        if (h < G && touches) {
          const float* pp = part + ((size_t)(tid + gi) * G + h) * GA_PART;
          pm[h] = __ldcg(pp + D); pl[h] = __ldcg(pp + D + 1);
        }
      }
#pragma unroll
      for (int h = 0; h < RBQ_MAX_G; ++h) {
        float v = pm[h];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) s_red[h * GA_WARPS + warp] = v;
      }
      __syncthreads();
      float mall[RBQ_MAX_G];
#pragma unroll
      for (int h = 0; h < RBQ_MAX_G; ++h) {
        float v = -INFINITY;
#pragma unroll
        for (int w = 0; w < GA_WARPS; ++w) v = fmaxf(v, s_red[h * GA_WARPS + w]);
        mall[h] = v;
        const float f = (pm[h] == -INFINITY) ? 0.0f : exp2f(pm[h] - v);
        s_f[h * GA_THREADS + tid] = f;
        float fl = f * pl[h];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) fl += __shfl_xor_sync(0xffffffffu, fl, o);
        if (lane == 0) s_red[(RBQ_MAX_G + h) * GA_WARPS + warp] = fl;
      }
      __syncthreads();
      const int item = tid % ITEMS, half = tid / ITEMS, d4 = (item % TPH) * 4;
      const int h = (half < NH) ? (item / TPH) : RBQ_MAX_G;     // threads beyond NH * ITEMS only take part in the barriers
      float mm = -INFINITY;
#pragma unroll
      for (int hh = 0; hh < RBQ_MAX_G; ++hh) mm = (hh == h) ? mall[hh] : mm;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float ll = 0.0f;
      if (h < G) {
        const float* pcol = part + ((size_t)gi * G + h) * GA_PART + d4;
        const size_t pstride = (size_t)G * GA_PART;
        constexpr int MU = 24;                                  // slot partials in flight per thread: one round for <= 48 slots
        for (int c0 = clo + half; c0 <= chi; c0 += MU * NH) {
          float f[MU];
          float4 v[MU];
#pragma unroll
          for (int k = 0; k < MU; ++k) {
            const int c = c0 + NH * k;
            f[k] = (c <= chi) ? s_f[h * GA_THREADS + c] : 0.0f;
            v[k] = (f[k] != 0.0f) ? __ldcg(reinterpret_cast<const float4*>(pcol + (size_t)c * pstride)) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
#pragma unroll
          for (int k = 0; k < MU; ++k) {
            acc.x = fmaf(f[k], v[k].x, acc.x); acc.y = fmaf(f[k], v[k].y, acc.y);
            acc.z = fmaf(f[k], v[k].z, acc.z); acc.w = fmaf(f[k], v[k].w, acc.w);
          }
        }
#pragma unroll
        for (int w = 0; w < GA_WARPS; ++w) ll += s_red[(RBQ_MAX_G + h) * GA_WARPS + w];
      }
      if (half >= 1 && half < NH) s_o[(half - 1) * ITEMS + item] = acc;
      __syncthreads();
      if (half == 0 && h < G) {
#pragma unroll
        for (int k = 1; k < NH; ++k) {
          const float4 o2 = s_o[(k - 1) * ITEMS + item];
          acc.x += o2.x; acc.y += o2.y; acc.z += o2.z; acc.w += o2.w;
        }
        const bool empty = !(ll > 0.0f);
        const float inv = empty ? 0.0f : 1.0f / ll;
        const size_t orow = (size_t)b * Hq + (size_t)g * G + h;
        const float r4[4] = {acc.x * inv, acc.y * inv, acc.z * inv, acc.w * inv};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (out_bf16) reinterpret_cast<__nv_bfloat16*>(out)[orow * D + d4 + k] = __float2bfloat16_rn(r4[k]);
          else reinterpret_cast<float*>(out)[orow * D + d4 + k] = r4[k];
        }
        if (lse && d4 == 0) lse[orow] = empty ? -INFINITY : mm * 0.6931471805599453f + logf(ll);
      }
      if (tid == 0) gdone[gi] = 0;                             // ready for the next step
      if (tid == 0) RBQ_STAMP(gather_probe, 8);
    }
    __syncthreads();                                           // staging area free before the next group's pipeline
  }
}

// ---- gather attention straight from the selection bitmaps (no plan kernel, no union list in global memory) ----------------
// The union of a KV group's G selection bitmaps is expanded where it is consumed.  Work unit: a CLAIM of 1 .. GB_CW
// consecutive bitmap words (32 tokens each) of one group, all G rows; the pending-window rows follow the bitmap words as
// words of 32 rows.  A warp expands a claim into its private ring of entries (token | head mask << 28) in shared memory
// (dense groups: one word per step, lane = token; sparse groups: all words of the claim at once, lane = one byte of one word);
// its cp.async pipeline takes 16-entry tiles from the ring and runs on across claim boundaries.
//   * across groups the CTAs are placed by the groups' COSTS = union rows + tokens / RBQ_GB_TOKDIV (sparse groups stream
//     slower per row: more bitmap to scan, isolated 512-byte rows) + RBQ_GB_PEN (every visit of a group costs a prologue, a
//     pipeline drain, a merge and an arrival), the union size being an estimate (build_cost_table):
//     equal contiguous ranges of the concatenated costs, one per CTA, boundaries snapped to the borders of large groups.  A
//     wrong estimate costs balance only, never correctness;
//   * inside a group the words are handed out dynamically: one atomicAdd per claim on the group's counter, issued one claim
//     ahead so that its latency and that of the bitmap words hide behind the tiles in flight; guided sizes (GB_CW0 .. 8 words
//     = ~64 rows while plenty is left, one word at the end of the group); the first claim of every warp of the CTAs that START
//     in the group is static, so no atomic sits in front of the first tile;
//   * every CTA whose range touches a group arrives at it (possibly with an empty partial); the last one merges the partials
//     into out / lse, stores the group's exact-to-estimated union ratio for the next step and resets the counters.
// The accumulation order of a group's rows therefore depends on the hand-out: results are reproducible to rounding (~1e-6
// relative), not bit for bit; RBQ_GATHER_PLAN=1 selects the static plan + union-list path below, which is.
// Measured at config 2 (stage events): plan 10.3 us + gather 55.2 us -> 56.3 us; step 90.9 -> 82.8 us (profiles/r02_ncu.md).
constexpr int GB_CW = 8;                                     // bitmap words (32 tokens each) per claim at most: one word per lane and head
constexpr int GB_CW0 = 4;                                    // words of a warp's static first claim
constexpr int GB_RING = 512;                                 // entries per warp ring (>= 15 left over + one claim)
#ifndef RBQ_GB_TOKDIV
#define RBQ_GB_TOKDIV 14                                     // cost of a group = union rows + tokens / RBQ_GB_TOKDIV (scan + sparse-row penalty)
#endif
#ifndef RBQ_GB_PEN
#define RBQ_GB_PEN 800                                       // fixed cost of a group (one visit: prologue, drain, merge, arrival) in row units
#endif
#ifndef RBQ_GB_BYTEPAR
#define RBQ_GB_BYTEPAR 5                                     // n > 0: byte-parallel expansion of the claims of groups whose claims exceed n words (see fill)
#endif
#ifndef RBQ_GB_SNAP
#define RBQ_GB_SNAP 6                                        // CTA boundaries snap to boundaries between groups worth >= this many CTAs each
#endif

// s_start[gi] = sum over groups < gi of the groups' costs; every CTA computes the same table.  The size of a group's union is
// not known when S7 starts (S6 leaves per-row counts); it is ESTIMATED as rho_g * n (1 - prod_h (1 - cnt_h / n)): the size G
// independent selections of these counts would have, times the ratio rho_g = exact / independent that this kernel measured
// for the same group in the previous step (the heads of a group correlate through the keys they share; the ratio is a
// property of the group much more than of the query).  0 = no history yet: 1.  A wrong estimate costs balance only.
__device__ void build_cost_table(const int32_t* __restrict__ sel_cnt, const float* __restrict__ rho, const int32_t* __restrict__ n_indexed,
                                 const int32_t* __restrict__ n_total, int ngroups, int Hq, int Hkv, int* s_start, int* s_warp,
                                 int nthreads, int* s_nidx, int* s_npend, float* s_ind) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
  const int G = Hq / Hkv;
  const int per = (ngroups + nthreads - 1) / nthreads;
  const int g0 = tid * per;
  int local = 0;
  for (int gi = g0; gi < min(ngroups, g0 + per); ++gi) {
    const int b = gi / Hkv, g = gi % Hkv;
    const int ni = max(0, n_indexed[b]), np = max(0, n_total[b] - ni);
    int cnt[RBQ_MAX_G];
#pragma unroll
    for (int h = 0; h < RBQ_MAX_G; ++h) cnt[h] = (h < G) ? __ldcg(sel_cnt + (size_t)b * Hq + (size_t)g * G + h) : 0;
    const float r = __ldcg(rho + gi);
    int est = 0;
    float ind = 0.0f;
    if (ni > 0) {
      const float inv = 1.0f / (float)ni;
      float keep = 1.0f;
      int mx = 0;
      long long sum = 0;
#pragma unroll
      for (int h = 0; h < RBQ_MAX_G; ++h) {
        const int c = min(max(cnt[h], 0), ni);
        keep *= 1.0f - (float)c * inv;
        mx = max(mx, c);
        sum += c;
      }
      ind = (float)ni * (1.0f - keep);
      est = (int)(ind * (r > 0.0f ? r : 1.0f) + 0.5f);
      est = min(max(est, mx), (int)min((long long)ni, sum));
    }
    const int cost = (est + np > 0) ? est + np + ni / RBQ_GB_TOKDIV + RBQ_GB_PEN : 0;   // rows + scanning the bitmaps of ni tokens + one visit
    s_nidx[gi] = ni;
    s_npend[gi] = np;
    s_ind[gi] = ind;
    s_start[gi] = cost;                                       // the group's own cost for now, its prefix below
    local += cost;
  }
  int incl = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int woff = 0, total = 0;
  for (int w = 0; w < nwarps; ++w) { if (w < warp) woff += s_warp[w]; total += s_warp[w]; }
  int run = woff + incl - local;
  for (int gi = g0; gi < min(ngroups, g0 + per); ++gi) {
    const int v = s_start[gi];
    s_start[gi] = run;
    run += v;
  }
  if (tid == 0) s_start[ngroups] = total;
  __syncthreads();
}

// CTA boundaries in the cost space, snapped: s_bound[c] = floor(total c / nce), and the boundary nearest to the border
// between two groups worth >= RBQ_GB_SNAP CTA shares each moves onto that border if it is less than half a share away, so
// that large groups get whole CTAs (a CTA that straddles two groups pays a second prologue and merge at the very end of the
// kernel; inside a group the work is shared dynamically anyway, so the price is an imbalance of at most half a CTA in
// RBQ_GB_SNAP).  Strictly increasing in c (two boundaries a share apart cannot both be closer than half a share to one
// border); identical in every CTA.
__device__ void build_bounds(const int* s_start, int ngroups, unsigned total, int nce, int* s_bound, int nthreads) {
  const int tid = threadIdx.x;
  const unsigned q0 = total / (unsigned)nce, r0 = total - q0 * (unsigned)nce;   // floor(total c / nce) = q0 c + floor(r0 c / nce)
  for (int c = tid; c <= nce; c += nthreads) s_bound[c] = (c >= nce) ? (int)total : (int)(q0 * (unsigned)c + (r0 * (unsigned)c) / (unsigned)nce);
  __syncthreads();
  const int share = (int)q0;
  const float c_per_cost = (float)nce / (float)total;
  for (int k = 1 + tid; k < ngroups; k += nthreads) {
    const int bnd = s_start[k];
    const long long big = (long long)RBQ_GB_SNAP * share;
    if ((long long)bnd - s_start[k - 1] < big || (long long)s_start[k + 1] - bnd < big) continue;
    int c = (int)((float)bnd * c_per_cost + 0.5f);             // nearest boundary, up to rounding: look at its neighbours too
    c = min(max(c, 1), nce - 1);
    int best = -1, bd = 0x7fffffff;
    for (int cc = max(1, c - 1); cc <= min(nce - 1, c + 1); ++cc) {   // (no other border is near enough to move these three)
      const int x = s_bound[cc], dist = x > bnd ? x - bnd : bnd - x;
      if (dist < bd) { bd = dist; best = cc; }
    }
    if (best > 0 && 2 * bd < share) s_bound[best] = bnd;
  }
  __syncthreads();
}

// grid = number of SMs (persistent), GA_THREADS threads, GaCfg<D>::SMEM dynamic shared memory.
// part: [gridDim.x + ngroups][G][GA_PART]; the partial of (CTA c, group gi) lives in slot c + gi.
// gnext / gdone: [ngroups], zero on entry, zero again on exit.
template <int D>
__global__ void __launch_bounds__(GA_THREADS, 1)
attn_gather_bits_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ K, const __nv_bfloat16* __restrict__ V,
                        long long sb, long long sh, long long st, const uint32_t* __restrict__ bits, int wpr,
                        const int32_t* __restrict__ sel_cnt, float* __restrict__ rho, int32_t* __restrict__ uexact,
                        const int32_t* __restrict__ n_indexed,
                        const int32_t* __restrict__ n_total, int ngroups, int Hq, int Hkv, float scale_log2,
                        float* __restrict__ part, int32_t* __restrict__ gdone, int32_t* __restrict__ gnext,
                        void* __restrict__ out, int out_bf16, float* __restrict__ lse) {
  using C = GaCfg<D>;
  constexpr int GA_TILE_BYTES = C::TILE_BYTES, GA_STAGE_BYTES = C::STAGE_BYTES, GA_PART = C::PART, RB = C::ROW_BYTES, CPR = C::CPR;
  constexpr int LSH = (D == 64) ? 3 : 4;                       // log2(CPR)
  extern __shared__ __align__(128) unsigned char ga_smem[];
  __shared__ int s_start[AT_MAX_GROUPS + 1], s_nidx[AT_MAX_GROUPS], s_npend[AT_MAX_GROUPS];
  __shared__ uint32_t s_ring[GA_WARPS][GB_RING];
  __shared__ int s_bound[GA_THREADS + 1];                     // snapped CTA boundaries in the cost space
  __shared__ float s_ind[AT_MAX_GROUPS];                      // union size of independent selections (the estimate before rho)
  __shared__ int s_rows;                                      // entries this CTA expanded in the current group
  __shared__ int s_warp[GA_WARPS];
  __shared__ int s_last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g4 = lane >> 2, t4 = lane & 3;                    // MMA fragment coordinates
  const int G = Hq / Hkv;
  if (tid == 0) RBQ_STAMP(gather_probe, 0);
#ifdef RBQ_PROBE
  if (tid == 0 && blockIdx.x < RBQ_PROBE_CTAS) { gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 13] = 0; gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 14] = 0; }
  __syncthreads();
#endif
  rbq_pdl_wait();                                             // selection bitmaps and counts of S6
  if (tid == 0) { RBQ_STAMP(gather_probe, 1); s_rows = 0; }    // (barriers inside the table builders below)

  build_cost_table(sel_cnt, rho, n_indexed, n_total, ngroups, Hq, Hkv, s_start, s_warp, GA_THREADS, s_nidx, s_npend, s_ind);
  if (tid == 0) RBQ_STAMP(gather_probe, 2);
  const unsigned total = (unsigned)s_start[ngroups];
  if (blockIdx.x == 0) {                                      // groups with nothing to attend: out = 0, lse = -inf
    for (int gq = 0; gq < ngroups; ++gq) {
      if (s_start[gq + 1] != s_start[gq]) continue;
      for (int hd = tid; hd < G * D; hd += GA_THREADS) {
        const size_t orow = (size_t)(gq / Hkv) * Hq + (size_t)(gq % Hkv) * G + hd / D;
        if (out_bf16) reinterpret_cast<__nv_bfloat16*>(out)[orow * D + hd % D] = __float2bfloat16_rn(0.0f);
        else reinterpret_cast<float*>(out)[orow * D + hd % D] = 0.0f;
        if (lse && hd % D == 0) lse[orow] = -INFINITY;
      }
    }
  }
  const int nce = (int)min((unsigned)gridDim.x, total);       // CTAs with a non-empty range
  if ((int)blockIdx.x >= nce) return;
  build_bounds(s_start, ngroups, total, nce, s_bound, GA_THREADS);
  const float c_per_cost = (float)nce / (float)total;
  const int r0 = s_bound[blockIdx.x], r1 = s_bound[blockIdx.x + 1];
  if (r0 >= r1) return;
  int gi = 0;                                                 // first group with s_start[gi + 1] > r0
  {
    int lo = 0, hi = ngroups - 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (s_start[mid + 1] > r0) hi = mid; else lo = mid + 1;
    }
    gi = lo;
  }
  if (tid == 0) RBQ_STAMP(gather_probe, 9);
  unsigned char* my_smem = ga_smem + (size_t)warp * GA_STAGES * GA_STAGE_BYTES;
  const uint32_t my_base = smem_u32(my_smem);
  uint32_t* ring = s_ring[warp];
  const unsigned lt = (1u << lane) - 1u;

  for (; gi < ngroups && s_start[gi] < r1; ++gi) {
    const int ga = s_start[gi], gb = s_start[gi + 1];
    if (ga >= gb) continue;
    const int b = gi / Hkv, g = gi % Hkv;
    const int nidx = s_nidx[gi], npend = s_npend[gi];
    // A operand: Q rows of the group's heads (rows >= G are zero); requested first, used after the claim set-up below
    uint32_t qa[D / 16][2];
    {
      const uint32_t* qp = reinterpret_cast<const uint32_t*>(q + ((size_t)b * Hq + (size_t)g * G + min(g4, G - 1)) * D);
#pragma unroll
      for (int ks = 0; ks < D / 16; ++ks) {
        qa[ks][0] = (g4 < G) ? qp[8 * ks + t4] : 0u;
        qa[ks][1] = (g4 < G) ? qp[8 * ks + 4 + t4] : 0u;
      }
    }
    // CTAs whose range touches [ga, gb): clo = last c with s_bound[c] <= ga, chi = last c with s_bound[c] < gb (the bounds are
    // strictly increasing and within half a share of total c / nce: a guess and a short walk)
    int clo = min(max((int)((float)ga * c_per_cost), 0), nce - 1);
    while (clo < nce - 1 && s_bound[clo + 1] <= ga) ++clo;
    while (clo > 0 && s_bound[clo] > ga) --clo;
    int chi = min(max((int)((float)gb * c_per_cost), 0), nce - 1);
    while (chi < nce - 1 && s_bound[chi + 1] < gb) ++chi;
    while (chi > 0 && s_bound[chi] >= gb) --chi;
    const int cfl = (s_bound[clo] >= ga) ? clo : clo + 1;
    const int nw = (nidx + 31) >> 5;                           // bitmap words; pending rows follow as words of 32 rows
    const int nwt = nw + ((npend + 31) >> 5);
    const int nwg = max(1, chi - clo + 1) * GA_WARPS;          // warps that share the group
    const int dyn_base = max(0, chi - cfl + 1) * GA_WARPS * GB_CW0;   // words below it are the static first claims
    // words per claim: ~64 attended rows while plenty is left, down to one word at the end of the group
    const int cw_max = min(GB_CW, max(GB_CW0, (int)(2.0f * (float)max(nidx, 1) / (float)max(gb - ga, 1))));
#if RBQ_GB_BYTEPAR
    const bool bytepar = cw_max > RBQ_GB_BYTEPAR;              // warp-uniform, per group
#endif
    const __nv_bfloat16* Kb = K + (long long)b * sb + (long long)g * sh;
    const __nv_bfloat16* Vb = V + (long long)b * sb + (long long)g * sh;
    // lane l loads word (l & 7) of head (l >> 3) of a claim
    const uint32_t* wsrc = bits + ((size_t)b * Hq + (size_t)g * G + min(lane >> 3, G - 1)) * wpr + (lane & 7);
    const bool wlane = (lane >> 3) < G;
    int32_t* cnt_ptr = gnext + gi;
    // The last CTA of a group whose range runs on into the next group takes only its share of this one (per warp, in cost
    // units) and moves on: what it leaves is picked up by the CTAs that end in the group.  Without the limit a CTA that is
    // alone in a small group at first (its neighbour still busy with its own first group) would take all of it.
    const bool leave_early = (int)blockIdx.x == chi && chi > clo && r1 > gb;
    const int limit = leave_early ? max(1, (gb - max(r0, ga)) / GA_WARPS) : 0x7fffffff;
    int consumed = RBQ_GB_PEN / GA_WARPS;                      // this visit's own fixed cost counts towards the share

    if (tid == 0) RBQ_STAMP(gather_probe, 12);
    // claim stream of this warp: [w_a, w_a + n_a) = words to expand next (bitmap words in pre_a); raw_b / n_b = the claim after
    int w_a, n_a, raw_b = 0, n_b = 0;
    uint32_t pre_a = 0u;
    auto load_words = [&](int w0, int n) -> uint32_t {
      return (wlane && (lane & 7) < n && w0 + (lane & 7) < nw) ? __ldcg(wsrc + w0) : 0u;
    };
    auto claim_size = [&](int from) -> int {                  // guided: half of an even share of what is left, 1 .. cw_max words
      return max(1, min(cw_max, (nwt - from) / (2 * nwg)));
    };
    if ((int)blockIdx.x >= cfl) {
      w_a = (((int)blockIdx.x - cfl) * GA_WARPS + warp) * GB_CW0;
      n_a = GB_CW0;
    } else {                                                   // second or later group of this CTA: every claim dynamic
      n_a = cw_max;
      int v = 0;
      if (lane == 0) v = atomicAdd(cnt_ptr, n_a);
      w_a = dyn_base + __shfl_sync(0xffffffffu, v, 0);
    }
    n_a = max(0, min(n_a, nwt - w_a));
    if (n_a > 0) {
      pre_a = load_words(w_a, n_a);
      n_b = claim_size(w_a);
      if (lane == 0) raw_b = atomicAdd(cnt_ptr, n_b);
    }
    if (tid == 0) RBQ_STAMP(gather_probe, 10);
    float m_run = -INFINITY, l_run = 0.0f;
    float o[D / 8][4];
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt) { o[nt][0] = 0.0f; o[nt][1] = 0.0f; o[nt][2] = 0.0f; o[nt][3] = 0.0f; }

    int head = 0, tail = 0;                                    // ring positions (monotone; slot = position & (GB_RING - 1))
    // expand claims until a whole tile is available or the group's words are exhausted
    auto fill = [&]() {
      while (tail - head < GA_TILE && n_a > 0) {
        consumed += (n_a * 32) / RBQ_GB_TOKDIV - tail;
#if RBQ_GB_BYTEPAR
        // sparse groups (claims of more than RBQ_GB_BYTEPAR words): all bitmap words of the claim at once: lane 4 j + s owns byte s of word j (8 tokens): the four heads' bytes side by
        // side in P, a warp scan of the bytes' popcounts, then every lane writes its <= 8 entries (head mask of bit b =
        // bits b, 8 + b, 16 + b, 24 + b of P, moved to bits 28 .. 31 by one multiplication)
        const int nbw = bytepar ? min(n_a, nw - w_a) : 0;
        if (nbw > 0) {
          const int j = lane >> 2, sB = lane & 3;
          const uint32_t w0 = __shfl_sync(0xffffffffu, pre_a, j), w1 = __shfl_sync(0xffffffffu, pre_a, 8 + j);
          const uint32_t w2 = __shfl_sync(0xffffffffu, pre_a, 16 + j), w3 = __shfl_sync(0xffffffffu, pre_a, 24 + j);
          const uint32_t selr = (uint32_t)sB | ((uint32_t)(4 + sB) << 4);
          const uint32_t P = __byte_perm(__byte_perm(w0, w1, selr), __byte_perm(w2, w3, selr), 0x5410);
          uint32_t u8 = (P | (P >> 8) | (P >> 16) | (P >> 24)) & 0xFFu;
          const int cnt = __popc(u8);
          int incl = cnt;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
          }
          const int tot = __shfl_sync(0xffffffffu, incl, 31);
          int pos = tail + incl - cnt;
          const uint32_t tokb = (uint32_t)((w_a + j) * 32 + 8 * sB);
          while (u8) {
            const int bp = __ffs(u8) - 1;
            u8 &= u8 - 1u;
            ring[pos & (GB_RING - 1)] = (tokb + (uint32_t)bp) | ((((P >> bp) & 0x01010101u) * 0x10204080u) & 0xF0000000u);
            ++pos;
          }
          __syncwarp();
          tail += tot;
        }
        for (int k = max(nbw, 0); k < n_a; ++k) {
#else
        for (int k = 0; k < n_a; ++k) {
#endif
          const int w = w_a + k;
          if (w < nw) {
            uint32_t u = 0u, mask = 0u;
#pragma unroll
            for (int h = 0; h < RBQ_MAX_G; ++h) {
              const uint32_t hwv = __shfl_sync(0xffffffffu, pre_a, 8 * h + k);
              u |= hwv;
              mask |= ((hwv >> lane) & 1u) << h;
            }
            if ((u >> lane) & 1u) ring[(tail + __popc(u & lt)) & (GB_RING - 1)] = (uint32_t)(w * 32 + lane) | (mask << 28);
            tail += __popc(u);
          } else {                                             // pending-window rows: attended by every head
            const int pr = (w - nw) * 32 + lane, pc = min(32, npend - (w - nw) * 32);
            if (lane < pc) ring[(tail + lane) & (GB_RING - 1)] = (uint32_t)(nidx + pr) | (0xFu << 28);
            tail += pc;
          }
        }
        consumed += tail;
        w_a = dyn_base + __shfl_sync(0xffffffffu, raw_b, 0);   // claimed one claim ago
        n_a = max(0, min(n_b, nwt - w_a));
        if (n_a > 0) {
          pre_a = load_words(w_a, n_a);
          n_b = (consumed < limit) ? claim_size(w_a) : 0;      // share taken: this claim is the last
          if (n_b > 0 && lane == 0) raw_b = atomicAdd(cnt_ptr, n_b);
        }
        __syncwarp();
      }
    };
    auto issue = [&](int i, uint32_t ent) {
      const uint32_t sbase = my_base + (uint32_t)((i % GA_STAGES) * GA_STAGE_BYTES);
#pragma unroll
      for (int k = 0; k < GA_TILE * CPR / 32; ++k) {           // 32 lanes cover 32 / CPR rows per step
        const int row = (32 / CPR) * k + (lane >> LSH), ch = lane & (CPR - 1);
        const uint32_t re = __shfl_sync(0xffffffffu, ent, row);
        const long long off = (long long)(re & 0x0FFFFFFFu) * st + ch * 8;
        const uint32_t d = sbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4));
        cp_async16(d, Kb + off);
        cp_async16(d + GA_TILE_BYTES, Vb + off);
      }
    };
    uint32_t ent_ring[GA_STAGES - 1];
#pragma unroll
    for (int s = 0; s < GA_STAGES - 1; ++s) ent_ring[s] = 0u;
    int issued = 0;
    for (int i = -(GA_STAGES - 1);; ++i) {
      fill();
      const int avail = tail - head;                           // >= GA_TILE, or what is left of an exhausted group
      uint32_t ent_new = 0u;
      if (avail > 0) {
        if (lane < GA_TILE && lane < avail) ent_new = ring[(head + lane) & (GB_RING - 1)];
        head += min(GA_TILE, avail);
        issue(issued, ent_new);
        ++issued;
      }
      cp_async_commit();
      const uint32_t ent = ent_ring[0];
#pragma unroll
      for (int s = 0; s + 1 < GA_STAGES - 1; ++s) ent_ring[s] = ent_ring[s + 1];
      ent_ring[GA_STAGES - 2] = ent_new;
      if (i < 0) continue;
      if (i >= issued) break;
      cp_async_wait<GA_STAGES - 1>();
      __syncwarp();
      if (tid == 0 && i == 0) RBQ_STAMP(gather_probe, 4);
      const uint32_t kbase = my_base + (uint32_t)((i % GA_STAGES) * GA_STAGE_BYTES), vbase = kbase + GA_TILE_BYTES;

      // S = Q K^T : two n-tiles of 8 tokens
      float s[2][4];
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        s[nt][0] = 0.0f; s[nt][1] = 0.0f; s[nt][2] = 0.0f; s[nt][3] = 0.0f;
        const int row = nt * 8 + (lane & 7);
#pragma unroll
        for (int j = 0; j < D / 32; ++j) {
          uint32_t bf[4];
          const int ch = 4 * j + (lane >> 3);
          ldsm_x4(bf, kbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4)));
          mma_bf16(s[nt], qa[2 * j][0], 0u, qa[2 * j][1], 0u, bf[0], bf[1]);
          mma_bf16(s[nt], qa[2 * j + 1][0], 0u, qa[2 * j + 1][1], 0u, bf[2], bf[3]);
        }
      }
      // head masks, online softmax (row = head g4; this lane: tokens nt*8 + 2*t4, +1)
      float tmax = -INFINITY;
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const uint32_t e0 = __shfl_sync(0xffffffffu, ent, nt * 8 + 2 * t4);
        const uint32_t e1 = __shfl_sync(0xffffffffu, ent, nt * 8 + 2 * t4 + 1);
        const bool ok0 = (e0 >> (28 + (g4 & 3))) & 1u, ok1 = (e1 >> (28 + (g4 & 3))) & 1u;
        s[nt][0] = (ok0 && g4 < G) ? s[nt][0] * scale_log2 : -INFINITY;
        s[nt][1] = (ok1 && g4 < G) ? s[nt][1] * scale_log2 : -INFINITY;
        tmax = fmaxf(tmax, fmaxf(s[nt][0], s[nt][1]));
      }
      tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
      tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
      const float m_new = fmaxf(m_run, tmax);
      const float m_use = (m_new == -INFINITY) ? 0.0f : m_new;
      const float resc = exp2f(m_run - m_use);                 // m_run = -inf -> 0
      m_run = m_new;
      const float p00 = exp2f(s[0][0] - m_use), p01 = exp2f(s[0][1] - m_use);
      const float p10 = exp2f(s[1][0] - m_use), p11 = exp2f(s[1][1] - m_use);
      l_run = l_run * resc + ((p00 + p01) + (p10 + p11));
      // P as bf16 hi + lo parts (two MMAs per V tile): keeps ~16 mantissa bits of the probabilities
      const uint32_t pa0 = pack_bf16(p00, p01), pa2 = pack_bf16(p10, p11);
      const uint32_t pb0 = pack_bf16(p00 - rbq_bf16lo(pa0), p01 - rbq_bf16hi(pa0));
      const uint32_t pb2 = pack_bf16(p10 - rbq_bf16lo(pa2), p11 - rbq_bf16hi(pa2));
      // O = O * resc + P V
#pragma unroll
      for (int c2 = 0; c2 < D / 16; ++c2) {
        uint32_t bf[4];
        const int row = (lane & 7) + ((lane >> 3) & 1) * 8, ch = 2 * c2 + (lane >> 4);
        ldsm_x4_t(bf, vbase + (uint32_t)(row * RB + ((ch ^ (row & 7)) << 4)));
        o[2 * c2][0] *= resc; o[2 * c2][1] *= resc;
        o[2 * c2 + 1][0] *= resc; o[2 * c2 + 1][1] *= resc;
        mma_bf16(o[2 * c2], pa0, 0u, pa2, 0u, bf[0], bf[1]);
        mma_bf16(o[2 * c2 + 1], pa0, 0u, pa2, 0u, bf[2], bf[3]);
        mma_bf16(o[2 * c2], pb0, 0u, pb2, 0u, bf[0], bf[1]);
        mma_bf16(o[2 * c2 + 1], pb0, 0u, pb2, 0u, bf[2], bf[3]);
      }
      __syncwarp();                                            // tile consumed before its stage is refilled
    }
    cp_async_wait<0>();
    rbq_pdl_trigger();                                        // dependents (the next step's S3) may become resident under the merge phase
    if (tid == 0) RBQ_STAMP(gather_probe, 5);
#ifdef RBQ_PROBE
    if (lane == 0 && blockIdx.x < RBQ_PROBE_CTAS) {
      atomicAdd(&gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 14], (unsigned long long)issued);
      if (warp == 0) { atomicAdd(&gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 13], 1ull << 32); atomicMax(&gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 13], (unsigned long long)gi | (gather_probe[blockIdx.x * RBQ_PROBE_SLOTS + 13] & ~0xFFFFull)); }
    }
#endif
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);

    // merge the warps of the CTA.  Every warp stages its partial in its OWN drained pipeline buffers (no barrier in front:
    // nobody else touches them), [G][GA_PART] floats at the start of the warp's region; s_rows is zero here (below)
    float* stg = reinterpret_cast<float*>(ga_smem);            // staging of warp w at stg + w * WSTG floats
    constexpr int WSTG = GA_STAGES * GA_STAGE_BYTES / 4;
    if (g4 < G) {
      float* dst = stg + (size_t)warp * WSTG + (size_t)g4 * GA_PART;
#pragma unroll
      for (int nt = 0; nt < D / 8; ++nt) { dst[8 * nt + 2 * t4] = o[nt][0]; dst[8 * nt + 2 * t4 + 1] = o[nt][1]; }
      if (t4 == 0) { dst[D] = m_run; dst[D + 1] = l_run; }
    }
    if (lane == 0 && tail > 0) atomicAdd(&s_rows, tail);       // every entry of the group is expanded exactly once, by some warp
    __syncthreads();
    if (tid == 0 && s_rows > 0) atomicAdd(&uexact[gi], s_rows);   // before this CTA's arrival (fence below)
    float* pdst = part + (size_t)(blockIdx.x + gi) * G * GA_PART;
    for (int idx = tid; idx < G * D; idx += GA_THREADS) {
      const int h = idx / D, d = idx % D;
      float mm = -INFINITY;
#pragma unroll
      for (int w = 0; w < GA_WARPS; ++w) mm = fmaxf(mm, stg[(size_t)w * WSTG + (size_t)h * GA_PART + D]);
      float oo = 0.0f, ll = 0.0f;
#pragma unroll
      for (int w = 0; w < GA_WARPS; ++w) {
        const float* sp = stg + (size_t)w * WSTG + (size_t)h * GA_PART;
        const float f = (sp[D] == -INFINITY) ? 0.0f : exp2f(sp[D] - mm);
        oo = fmaf(f, sp[d], oo);
        ll = fmaf(f, sp[D + 1], ll);
      }
      pdst[(size_t)h * GA_PART + d] = oo;
      if (d == 0) { pdst[(size_t)h * GA_PART + D] = mm; pdst[(size_t)h * GA_PART + D + 1] = ll; }
    }
    // ---- arrival: the last CTA that finishes a group merges the group's partials into out / lse -------------------------
    if (tid == 0) RBQ_STAMP(gather_probe, 6);
    __threadfence();
    const bool touches = tid >= clo && tid <= chi;
    const int expected = chi - clo + 1;
    __syncthreads();                                           // staging area free, partial stores fenced
    if (tid == 0) s_rows = 0;                                  // (read above, before this barrier; next used after the barriers below)
    if (tid == 0) s_last = (atomicAdd(&gdone[gi], 1) == expected - 1);
    __syncthreads();
    if (tid == 0) RBQ_STAMP(gather_probe, 7);
    if (s_last) {
      __threadfence();
      float* s_f = stg;                                        // [G][GA_THREADS]: factor 2^(m - max) of slot c
      constexpr int TPH = D / 4, ITEMS = RBQ_MAX_G * TPH;     // threads per head (4 dims each), (head, dim group) items
      constexpr int NH = GA_THREADS / ITEMS;                   // slot subsets worked on in parallel (2 at D = 128, 4 at D = 64)
      constexpr int MU = 24;                                    // slot partials in flight per thread: one round for <= 48 slots
      float4* s_o = reinterpret_cast<float4*>(stg + 2 * RBQ_MAX_G * GA_THREADS);   // [NH - 1][ITEMS] partial sums of subsets 1 ..
      // thread tid owns slot tid: per-head maximum and normaliser by block reductions (warp shuffles + one shared round)
      float* s_red = stg + 2 * RBQ_MAX_G * GA_THREADS + 4 * (NH > 1 ? (NH - 1) * ITEMS : 1);   // [2][RBQ_MAX_G][GA_WARPS]
      const int item = tid % ITEMS, half = tid / ITEMS, d4 = (item % TPH) * 4;
      const int h = (half < NH) ? (item / TPH) : RBQ_MAX_G;     // threads beyond NH * ITEMS only take part in the barriers
      const float* pcol = part + ((size_t)gi * G + min(h, G - 1)) * GA_PART + d4;
      const size_t pstride = (size_t)G * GA_PART;
      // the first round of partial sums is requested together with the (m, l) pairs: one L2 round trip instead of two on the
      // path of the last CTA (the accumulators of the streaming loop are dead: registers are free)
      float4 v0[MU];
#pragma unroll
      for (int k = 0; k < MU; ++k) {
        const int c = clo + half + NH * k;
        v0[k] = (h < G && c <= chi) ? __ldcg(reinterpret_cast<const float4*>(pcol + (size_t)c * pstride)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      float pm[RBQ_MAX_G], pl[RBQ_MAX_G];
#pragma unroll
      for (int hh = 0; hh < RBQ_MAX_G; ++hh) {
        pm[hh] = -INFINITY; pl[hh] = 0.0f;
        if (hh < G && touches) {
          const float* pp = part + ((size_t)(tid + gi) * G + hh) * GA_PART;
          pm[hh] = __ldcg(pp + D); pl[hh] = __ldcg(pp + D + 1);
        }
      }
#pragma unroll
      for (int hh = 0; hh < RBQ_MAX_G; ++hh) {
        float v = pm[hh];
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o2));
        if (lane == 0) s_red[hh * GA_WARPS + warp] = v;
      }
      __syncthreads();
      float mall[RBQ_MAX_G];
#pragma unroll
      for (int hh = 0; hh < RBQ_MAX_G; ++hh) {
        float v = -INFINITY;
#pragma unroll
        for (int w = 0; w < GA_WARPS; ++w) v = fmaxf(v, s_red[hh * GA_WARPS + w]);
        mall[hh] = v;
        const float f = (pm[hh] == -INFINITY) ? 0.0f : exp2f(pm[hh] - v);
        s_f[hh * GA_THREADS + tid] = f;
        float fl = f * pl[hh];
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) fl += __shfl_xor_sync(0xffffffffu, fl, o2);
        if (lane == 0) s_red[(RBQ_MAX_G + hh) * GA_WARPS + warp] = fl;
      }
      __syncthreads();
      float mm = -INFINITY;
#pragma unroll
      for (int hh = 0; hh < RBQ_MAX_G; ++hh) mm = (hh == h) ? mall[hh] : mm;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float ll = 0.0f;
      if (h < G) {
#pragma unroll
        for (int k = 0; k < MU; ++k) {                          // first round: already here
          const int c = clo + half + NH * k;
          const float f = (c <= chi) ? s_f[h * GA_THREADS + c] : 0.0f;   // an empty partial (f = 0) holds zeros
          acc.x = fmaf(f, v0[k].x, acc.x); acc.y = fmaf(f, v0[k].y, acc.y);
          acc.z = fmaf(f, v0[k].z, acc.z); acc.w = fmaf(f, v0[k].w, acc.w);
        }
        for (int c0 = clo + half + MU * NH; c0 <= chi; c0 += MU * NH) {   // groups shared by more than MU * NH CTAs
          float f[MU];
          float4 v[MU];
#pragma unroll
          for (int k = 0; k < MU; ++k) {
            const int c = c0 + NH * k;
            f[k] = (c <= chi) ? s_f[h * GA_THREADS + c] : 0.0f;
            v[k] = (f[k] != 0.0f) ? __ldcg(reinterpret_cast<const float4*>(pcol + (size_t)c * pstride)) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
#pragma unroll
          for (int k = 0; k < MU; ++k) {
            acc.x = fmaf(f[k], v[k].x, acc.x); acc.y = fmaf(f[k], v[k].y, acc.y);
            acc.z = fmaf(f[k], v[k].z, acc.z); acc.w = fmaf(f[k], v[k].w, acc.w);
          }
        }
#pragma unroll
        for (int w = 0; w < GA_WARPS; ++w) ll += s_red[(RBQ_MAX_G + h) * GA_WARPS + w];
      }
      if (half >= 1 && half < NH) s_o[(half - 1) * ITEMS + item] = acc;
      __syncthreads();
      if (half == 0 && h < G) {
#pragma unroll
        for (int k = 1; k < NH; ++k) {
          const float4 o2 = s_o[(k - 1) * ITEMS + item];
          acc.x += o2.x; acc.y += o2.y; acc.z += o2.z; acc.w += o2.w;
        }
        const bool empty = !(ll > 0.0f);
        const float inv = empty ? 0.0f : 1.0f / ll;
        const size_t orow = (size_t)b * Hq + (size_t)g * G + h;
        const float r4[4] = {acc.x * inv, acc.y * inv, acc.z * inv, acc.w * inv};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (out_bf16) reinterpret_cast<__nv_bfloat16*>(out)[orow * D + d4 + k] = __float2bfloat16_rn(r4[k]);
          else reinterpret_cast<float*>(out)[orow * D + d4 + k] = r4[k];
        }
        if (lse && d4 == 0) lse[orow] = empty ? -INFINITY : mm * 0.6931471805599453f + logf(ll);
      }
      if (tid == 0) {                                          // every touching CTA has made its last claim: ready for the next step
        gdone[gi] = 0; gnext[gi] = 0;
        const int ux = __ldcg(uexact + gi) - npend;            // exact size of the union (every arrival has added its entries)
        uexact[gi] = 0;
        const float ind = s_ind[gi];
        rho[gi] = (ind >= 1.0f && ux > 0) ? fminf(fmaxf((float)ux / ind, 0.05f), 4.0f) : 0.0f;
      }
      if (tid == 0) RBQ_STAMP(gather_probe, 8);
    }
    __syncthreads();                                           // staging area free before the next group's pipeline
  }
}

// ---- FP32-pipe kernel for fp32 K/V or q (parity config 0) and for head_dim 256: split-K over the group's union list ------
constexpr int AT_THREADS = 256;
constexpr int AT_WARPS = AT_THREADS / 32;
constexpr int AT_CHUNK = AT_WARPS * 32;       // union rows per chunk: one 32-row strip per warp

// N consecutive elements of a row as floats, in 4-element pieces (8-byte loads for bf16, 16-byte loads for fp32)
template <int N>
__device__ __forceinline__ void load_row(const __nv_bfloat16* p, float (&v)[N]) {
#pragma unroll
  for (int k = 0; k < N / 4; ++k) {
    const uint2 u = *reinterpret_cast<const uint2*>(p + 4 * k);
    v[4 * k] = rbq_bf16lo(u.x); v[4 * k + 1] = rbq_bf16hi(u.x); v[4 * k + 2] = rbq_bf16lo(u.y); v[4 * k + 3] = rbq_bf16hi(u.y);
  }
}
template <int N>
__device__ __forceinline__ void load_row(const float* p, float (&v)[N]) {
#pragma unroll
  for (int k = 0; k < N / 4; ++k) {
    const float4 a = *reinterpret_cast<const float4*>(p + 4 * k);
    v[4 * k] = a.x; v[4 * k + 1] = a.y; v[4 * k + 2] = a.z; v[4 * k + 3] = a.w;
  }
}

// grid = (max chunks per group, B*Hq rows).  Chunk ch of row (b,h) covers union rows [ch*256, ch*256+256) of the
// row's KV group; rows whose head-mask bit is clear are skipped.  part: [rows][max_chunks][D + 2] (o, m, l).
template <typename T, typename TQ, int D>
__global__ void __launch_bounds__(AT_THREADS)
attn_simt_kernel(const TQ* __restrict__ q, const T* __restrict__ K, const T* __restrict__ V, long long sb, long long sh,
                 long long st, const uint32_t* __restrict__ ulist, const int32_t* __restrict__ ucount,
                 const int32_t* __restrict__ n_indexed, const int32_t* __restrict__ n_total, int Hq, int Hkv, int Lcap,
                 float sm_scale, int max_chunks, float* __restrict__ part) {
  constexpr int AT_PART = D + 2, DPL = D / 16;                // dims per lane: a half-warp covers a row
  constexpr int NJ = DPL >= 16 ? 2 : 4;                       // rows per half-warp and step (register budget)
  __shared__ float s_part[AT_WARPS][AT_PART];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int half = lane >> 4, c = lane & 15;
  const int G = Hq / Hkv;
  const int row = blockIdx.y, b = row / Hq, h = row % Hq, g = h / G, hl = h % G;
  const int gi = b * Hkv + g;
  const int usel = ucount[gi], nidx = max(0, n_indexed[b]);
  const int na = usel + max(0, n_total[b] - nidx);
  const int ch = blockIdx.x;
  float* dst = part + ((size_t)row * max_chunks + ch) * AT_PART;
  if (ch * AT_CHUNK >= na) {
    if (tid == 0) { dst[D] = -INFINITY; dst[D + 1] = 0.0f; }
    return;
  }
  const int i0 = ch * AT_CHUNK + warp * 32;
  const int nw = max(0, min(32, na - i0));
  const T* Kb = K + (long long)b * sb + (long long)g * sh;
  const T* Vb = V + (long long)b * sb + (long long)g * sh;
  const uint32_t* ul = ulist + (size_t)gi * Lcap;

  float qv[DPL];
  {
    const TQ* qp = q + ((size_t)row * D + c * DPL);
#pragma unroll
    for (int d = 0; d < DPL; ++d) qv[d] = rbq_ld_elem(qp, d);
  }
  uint32_t my_ent = 0u;                                         // token | mask << 28 ; mask bit clear = not attended by this head
  if (lane < nw) {
    const int it = i0 + lane;
    my_ent = (it < usel) ? ul[it] : ((uint32_t)(nidx + (it - usel)) | (0xFu << 28));
  }
  float m = -INFINITY, l = 0.0f, acc[DPL];
#pragma unroll
  for (int d = 0; d < DPL; ++d) acc[d] = 0.0f;

  for (int base = 0; base < nw; base += 2 * NJ) {
    float kr[NJ][DPL], vr[NJ][DPL];
    bool ok[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int item = base + 2 * j + half;
      const uint32_t ent = __shfl_sync(0xffffffffu, my_ent, item & 31);
      ok[j] = (item < nw) && ((ent >> (28 + hl)) & 1u);
      const long long off = (long long)(ent & 0x0FFFFFFFu) * st + c * DPL;
      load_row<DPL>(Kb + off, kr[j]);                           // masked items read a valid row: harmless
      load_row<DPL>(Vb + off, vr[j]);
    }
    float s[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      float d0 = 0.0f;
#pragma unroll
      for (int d = 0; d < DPL; ++d) d0 = fmaf(qv[d], kr[j][d], d0);
      s[j] = d0;
    }
#pragma unroll
    for (int o = 8; o > 0; o >>= 1)
#pragma unroll
      for (int j = 0; j < NJ; ++j) s[j] += __shfl_xor_sync(0xffffffffu, s[j], o);
    float gmax = -INFINITY;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      s[j] = ok[j] ? s[j] * sm_scale : -INFINITY;
      gmax = fmaxf(gmax, s[j]);
    }
    gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, 16));
    const float m_new = fmaxf(m, gmax);
    const float m_use = (m_new == -INFINITY) ? 0.0f : m_new;
    const float resc = __expf(m - m_use);                       // m = -inf -> 0
    l *= resc;
#pragma unroll
    for (int d = 0; d < DPL; ++d) acc[d] *= resc;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const float p = __expf(s[j] - m_use);                     // masked: exp(-inf) = 0
      l += p;
#pragma unroll
      for (int d = 0; d < DPL; ++d) acc[d] = fmaf(p, vr[j][d], acc[d]);
    }
    m = m_new;
  }
  // merge the two half-warps (same m), then the warps of the CTA
  l += __shfl_xor_sync(0xffffffffu, l, 16);
#pragma unroll
  for (int d = 0; d < DPL; ++d) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], 16);
  if (half == 0) {
#pragma unroll
    for (int d = 0; d < DPL; ++d) s_part[warp][c * DPL + d] = acc[d];
    if (c == 0) { s_part[warp][D] = m; s_part[warp][D + 1] = l; }
  }
  __syncthreads();
  for (int d = tid; d < D; d += AT_THREADS) {
    float mm = -INFINITY;
#pragma unroll
    for (int w = 0; w < AT_WARPS; ++w) mm = fmaxf(mm, s_part[w][D]);
    float o = 0.0f, ll = 0.0f;
#pragma unroll
    for (int w = 0; w < AT_WARPS; ++w) {
      const float mw = s_part[w][D];
      const float f = (mw == -INFINITY) ? 0.0f : __expf(mw - mm);
      o = fmaf(f, s_part[w][d], o);
      ll = fmaf(f, s_part[w][D + 1], ll);
    }
    dst[d] = o;
    if (d == 0) { dst[D] = mm; dst[D + 1] = ll; }
  }
}

// grid = rows, D threads; natural-log units
template <typename TO>
__global__ void attn_simt_merge_kernel(const float* __restrict__ part, const int32_t* __restrict__ ucount, const int32_t* __restrict__ n_indexed,
                                       const int32_t* __restrict__ n_total, int Hq, int Hkv, int D, int max_chunks, TO* __restrict__ out,
                                       float* __restrict__ lse) {
  const int AT_PART = D + 2;
  const int row = blockIdx.x, d = threadIdx.x, b = row / Hq, G = Hq / Hkv;
  const int gi = b * Hkv + (row % Hq) / G;
  const int na = ucount[gi] + max(0, n_total[b] - max(0, n_indexed[b]));
  const int nch = min(max_chunks, (na + AT_CHUNK - 1) / AT_CHUNK);
  const float* base = part + (size_t)row * max_chunks * AT_PART;
  float mm = -INFINITY;
  for (int ch = 0; ch < nch; ++ch) mm = fmaxf(mm, base[(size_t)ch * AT_PART + D]);
  float o = 0.0f, l = 0.0f;
  for (int ch = 0; ch < nch; ++ch) {
    const float* p = base + (size_t)ch * AT_PART;
    const float f = (p[D] == -INFINITY) ? 0.0f : __expf(p[D] - mm);
    o = fmaf(f, p[d], o);
    l = fmaf(f, p[D + 1], l);
  }
  const bool empty = !(l > 0.0f);
  rbq_st_elem(out, (long long)row * D + d, empty ? 0.0f : o / l);
  if (lse && d == 0) lse[row] = empty ? -INFINITY : mm + logf(l);
}

template <typename T, typename TQ, int D>
int launch_simt_d(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const uint32_t* ulist, const int32_t* ucount,
                  int max_chunks, float* part, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  dim3 grid(max_chunks, rows);
  attn_simt_kernel<T, TQ, D><<<grid, AT_THREADS, 0, s>>>((const TQ*)q, (const T*)kv.k, (const T*)kv.v, kv.sb, kv.sh, kv.st, ulist,
                                                         ucount, idx->n_indexed, idx->n_total, ctx->cfg.n_q_heads,
                                                         ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, ctx->sm_scale, max_chunks, part);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
template <typename T, typename TQ>
int launch_simt(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const uint32_t* ulist, const int32_t* ucount,
                int max_chunks, float* part, cudaStream_t s) {
  switch (ctx->cfg.head_dim) {
    case 64: return launch_simt_d<T, TQ, 64>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
    case 256: return launch_simt_d<T, TQ, 256>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
    default: return launch_simt_d<T, TQ, 128>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
  }
}

}  // namespace

// tensor-pipe gather: bf16 K/V and q, head_dim 64 or 128 (256: 128 accumulator registers per thread would not fit)
static bool rbq_attention_uses_mma(const rbq_ctx* ctx) {
  return ctx->cfg.kv_dtype == RBQ_BF16 && ctx->cfg.q_dtype == RBQ_BF16 && ctx->cfg.head_dim <= 128;
}

bool rbq_attention_from_bits(const rbq_ctx* ctx) { return rbq_attention_uses_mma(ctx) && !ctx->gather_via_plan; }

template <int D>
static int launch_gather_d(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const uint32_t* ulist,
                           const int32_t* ucount, int groups, float* part, int32_t* gdone, void* out, float* lse, cudaStream_t s) {
  auto kern = attn_gather_kernel<D>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_GATHER + (D == 64 ? 0 : 1), kern, GaCfg<D>::SMEM);
  const int nc = min(ctx->sm_count, GA_THREADS);             // one persistent CTA per SM; the arrival count uses one thread per CTA
  RBQ_CUDA_OK(ctx, rbq_launch_pdl(kern, dim3(nc), dim3(GA_THREADS), (size_t)GaCfg<D>::SMEM, s, (const __nv_bfloat16*)q,
                                  (const __nv_bfloat16*)kv.k, (const __nv_bfloat16*)kv.v, kv.sb, kv.sh, kv.st,
                                  (const uint32_t*)ulist, (const int32_t*)ucount, (const int32_t*)idx->n_indexed,
                                  (const int32_t*)idx->n_total, groups, ctx->cfg.n_q_heads, ctx->cfg.n_kv_heads,
                                  ctx->cfg.max_tokens, ctx->sm_scale * 1.4426950408889634f, part, gdone, out,
                                  ctx->cfg.out_dtype == RBQ_BF16 ? 1 : 0, lse));
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

template <int D>
static int launch_gather_bits_d(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const uint32_t* bits, int wpr,
                                const int32_t* sel_cnt, float* rho, int32_t* uexact, int groups, float* part, int32_t* gdone, int32_t* gnext, void* out, float* lse,
                                cudaStream_t s) {
  auto kern = attn_gather_bits_kernel<D>;
  RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_GATHER + (D == 64 ? 2 : 3), kern, GaCfg<D>::SMEM);
  const int nc = min(ctx->sm_count, GA_THREADS);             // one persistent CTA per SM; the merge uses one thread per CTA
  RBQ_CUDA_OK(ctx, rbq_launch_pdl(kern, dim3(nc), dim3(GA_THREADS), (size_t)GaCfg<D>::SMEM, s, (const __nv_bfloat16*)q,
                                  (const __nv_bfloat16*)kv.k, (const __nv_bfloat16*)kv.v, kv.sb, kv.sh, kv.st, bits, wpr, sel_cnt, rho, uexact,
                                  (const int32_t*)idx->n_indexed, (const int32_t*)idx->n_total, groups, ctx->cfg.n_q_heads,
                                  ctx->cfg.n_kv_heads, ctx->sm_scale * 1.4426950408889634f, part, gdone, gnext, out,
                                  ctx->cfg.out_dtype == RBQ_BF16 ? 1 : 0, lse));
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

size_t rbq_attention_part_bytes(const rbq_ctx* ctx) {
  const size_t rows = (size_t)ctx->cfg.batch * ctx->cfg.n_q_heads, groups = (size_t)ctx->cfg.batch * ctx->cfg.n_kv_heads;
  const size_t D = ctx->cfg.head_dim;
  if (rbq_attention_uses_mma(ctx)) return ((size_t)ctx->sm_count + groups) * ctx->G * (D + 4) * sizeof(float);
  const size_t max_chunks = ((size_t)ctx->cfg.max_tokens + AT_CHUNK - 1) / AT_CHUNK;
  return rows * max_chunks * (D + 2) * sizeof(float);
}

int rbq_launch_bits_from_lists(rbq_ctx* ctx, const rbq_index* idx, const int32_t* sel_idx, const int32_t* sel_cnt, uint32_t* bits,
                               cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads;
  const int wpr = rbq_words_per_row(ctx);
  RBQ_CUDA_OK(ctx, cudaMemsetAsync(bits, 0, (size_t)rows * wpr * sizeof(uint32_t), s));
  dim3 grid(max(1, min(64, (ctx->cfg.max_tokens + 255) / 256)), rows);
  bits_from_lists_kernel<<<grid, 256, 0, s>>>(sel_idx, sel_cnt, idx->n_indexed, ctx->cfg.n_q_heads, ctx->cfg.max_tokens, wpr, bits);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

// S7 from the per-row selection bitmaps in the workspace: plan -> gather -> merge.
int rbq_launch_attention(rbq_ctx* ctx, const void* q, const RbqKV& kv, const rbq_index* idx, const uint32_t* bits,
                         const int32_t* sel_cnt, void* out, float* lse, cudaStream_t s) {
  const int rows = ctx->cfg.batch * ctx->cfg.n_q_heads, groups = ctx->cfg.batch * ctx->cfg.n_kv_heads;
  if (groups > AT_MAX_GROUPS) RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "batch*n_kv_heads %d > %d", groups, AT_MAX_GROUPS);
  const int wpr = rbq_words_per_row(ctx);
  char* ws = static_cast<char*>(ctx->ws);
  uint32_t* ulist = reinterpret_cast<uint32_t*>(ws + ctx->off_ulist);
  int32_t* ucount = reinterpret_cast<int32_t*>(ws + ctx->off_ucount);
  float* part = reinterpret_cast<float*>(ws + ctx->off_part);
  int32_t* gdone = reinterpret_cast<int32_t*>(ws + ctx->off_gdone);
  // bf16 tensor-pipe path: the gather expands the bitmaps itself (no plan launch, no union list)
  if (rbq_attention_from_bits(ctx)) {
    int32_t* gnext = reinterpret_cast<int32_t*>(ws + ctx->off_gnext);
    float* rho = reinterpret_cast<float*>(ws + ctx->off_rho);
    int32_t* uexact = reinterpret_cast<int32_t*>(ws + ctx->off_uexact);
    // (stage events: there is no plan stage on this path; rbq_profile_read reports 0 for it and does not read event 4)
    if (ctx->cfg.head_dim == 64)
      return launch_gather_bits_d<64>(ctx, q, kv, idx, bits, wpr, sel_cnt, rho, uexact, groups, part, gdone, gnext, out, lse, s);
    return launch_gather_bits_d<128>(ctx, q, kv, idx, bits, wpr, sel_cnt, rho, uexact, groups, part, gdone, gnext, out, lse, s);
  }
  int split = PL_MAX_SPLIT;
  while (split > 1 && (long long)groups * split > (long long)ctx->sm_count) split >>= 1;   // one wave at ONE CTA per SM (40-64 registers x 1 024 threads)
#define RBQ_PLAN_LAUNCH(SP)                                                                                          \
  RBQ_CUDA_OK(ctx, rbq_launch_pdl(attn_plan_kernel<SP>, dim3(SP, groups), dim3(PL_THREADS), 0, s, bits,                \
                                  (const int32_t*)idx->n_indexed, (const int32_t*)idx->n_total, ctx->cfg.n_q_heads,   \
                                  ctx->cfg.n_kv_heads, ctx->cfg.max_tokens, wpr, ulist, ucount, gdone))
  switch (split) {
    case 16: RBQ_PLAN_LAUNCH(16); break;
    case 8: RBQ_PLAN_LAUNCH(8); break;
    case 4: RBQ_PLAN_LAUNCH(4); break;
    case 2: RBQ_PLAN_LAUNCH(2); break;
    default: RBQ_PLAN_LAUNCH(1); break;
  }
  RBQ_LAUNCH_OK(ctx);
#undef RBQ_PLAN_LAUNCH
  if (ctx->stage_ev) RBQ_CUDA_OK(ctx, cudaEventRecord(ctx->stage_ev[4], s));
  const bool kbf = ctx->cfg.kv_dtype == RBQ_BF16, qbf = ctx->cfg.q_dtype == RBQ_BF16;
  if (rbq_attention_uses_mma(ctx)) {
    if (ctx->cfg.head_dim == 64) return launch_gather_d<64>(ctx, q, kv, idx, ulist, ucount, groups, part, gdone, out, lse, s);
    return launch_gather_d<128>(ctx, q, kv, idx, ulist, ucount, groups, part, gdone, out, lse, s);
  }
  const int max_chunks = (ctx->cfg.max_tokens + AT_CHUNK - 1) / AT_CHUNK;
  int rc;
  if (kbf && qbf) rc = launch_simt<__nv_bfloat16, __nv_bfloat16>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
  else if (kbf) rc = launch_simt<__nv_bfloat16, float>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
  else if (qbf) rc = launch_simt<float, __nv_bfloat16>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
  else rc = launch_simt<float, float>(ctx, q, kv, idx, ulist, ucount, max_chunks, part, s);
  if (rc != RBQ_OK) return rc;
  if (ctx->cfg.out_dtype == RBQ_BF16)
    attn_simt_merge_kernel<<<rows, ctx->cfg.head_dim, 0, s>>>(part, ucount, idx->n_indexed, idx->n_total, ctx->cfg.n_q_heads,
                                                              ctx->cfg.n_kv_heads, ctx->cfg.head_dim, max_chunks, (__nv_bfloat16*)out, lse);
  else
    attn_simt_merge_kernel<<<rows, ctx->cfg.head_dim, 0, s>>>(part, ucount, idx->n_indexed, idx->n_total, ctx->cfg.n_q_heads,
                                                              ctx->cfg.n_kv_heads, ctx->cfg.head_dim, max_chunks, (float*)out, lse);
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}

int rbq_probe_copy_gather(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, gather_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}

int rbq_probe_copy_plan(unsigned long long* host) {
#ifdef RBQ_PROBE
  if (cudaDeviceSynchronize() != cudaSuccess) return RBQ_ERR_CUDA;
  return cudaMemcpyFromSymbol(host, plan_probe, sizeof(unsigned long long) * RBQ_PROBE_CTAS * RBQ_PROBE_SLOTS) == cudaSuccess ? RBQ_OK : RBQ_ERR_CUDA;
#else
  (void)host;
  return RBQ_ERR_UNSUPPORTED;
#endif
}
