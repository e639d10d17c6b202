// rbq_qprep.cuh -- S3 as a device function: query pre-processing and INT4 quantisation of the G query heads of one
// (sequence, KV head) by a group of NT threads (Alg.2 lines 4-6, L168-172; Eq.5; L524; readings R1/R5/R6/R12
// of DESIGN.md).  Used by query_kernel (rbq_query.cu: the stand-alone S3 with its public outputs) and inside the
// estimator CTAs (rbq_estimate.cu: S3 fused into S4/S5, so that no separate launch sits in front of the code scan).
//
//   xq = q - c_q ; qn = ||xq||_2 ; u = xq/qn ; q' = u P (canonical fp32 order, as S1) ;
//   q_l = min q', q_r = max q', Delta = (q_r - q_l)/15 ; qu_j = clamp(floor((q'_j-q_l)/Delta + 1/2), 0, 15).
// Canonical order: ||xq||^2 and every q'_j are sequential fmaf chains, index ascending; the Walsh-Hadamard butterflies run
// level by level h = 1, 2, .., D/2 with (a, b) -> (a + b, a - b); the two fp64 dot products <q,c_k>, <c_q,c_k> are exact
// products summed by a fixed tree (32-lane xor tree per 32 dims, then a pairwise tree over the D/32 partials).
#pragma once
#include "rbq_common.cuh"

#ifndef RBQ_QPREP_STAMP          // timeline probes of the includer (probe build only)
#define RBQ_QPREP_STAMP(slot) do {} while (0)
#endif

template <int D>
struct __align__(16) RbqQPrepSmem {
  float x[RBQ_MAX_G][D];                    // xq, then u
  float y[RBQ_MAX_G][D];                    // q (for the fp64 dots), then q'
  float cq[RBQ_MAX_G][D];
  float ck[D];
  double dred[RBQ_MAX_G][2][D / 32];
  int isum[RBQ_MAX_G][D / 32];
  float qn[RBQ_MAX_G], ql[RBQ_MAX_G], delta[RBQ_MAX_G];
  uint8_t qu[RBQ_MAX_G][D];
};

// S3 for NP (1 or 2) pairs bg[0 .. NP) at once: the phases are chains of dependent latencies (global loads, a 128-long fmaf
// chain for the norm, another for every rotated coordinate), so a second pair interleaved with the first costs little more
// than one.  Results go to qc_out[p] (shared or global memory), scratch is sm[p].
// bar_id / nt: named barrier used by the nt participating threads (bar_id 0 with nt = blockDim.x is __syncthreads()).
// P_SMEM: the dense P is staged in shared memory at s_rot ([D][D]; a compile-time choice so that the reads stay LDS -- a
// pointer that may also be null makes the compiler fall back to generic loads); p_bar_sa != 0: shared address of the
// mbarrier (phase 0) on which that copy completes, awaited just before the rotation.  Otherwise P is read from `rot` (L2).
// qu_out / qparams / q_copy: optional public outputs (NP = 1 callers only pass them).
template <typename TQ, int D, int NP, bool P_SMEM>
__device__ __forceinline__ void rbq_qprep(const TQ* __restrict__ q, const float* __restrict__ c_q, const float* __restrict__ c_k,
                                          const float* __restrict__ rot, const float* s_rot, uint32_t p_bar_sa, int rot_kind, int Hq, int Hkv,
                                          const int (&bgs)[NP], const int (&rows0)[NP], float sm_scale, RbqQPrepSmem<D>* sm, int tid, int nt, int bar_id,
                                          RbqQConst* __restrict__ qc_out, uint8_t* __restrict__ qu_out,
                                          float* __restrict__ qparams, TQ* __restrict__ q_copy, int h_off = 0, int G_out = 0) {
  // Single-head mode (h_off, G_out given; the caller passes Hq == Hkv, so that G == 1 in here, and rows0[p] = the head's
  // own row): the caller works on head h_off of a group of G_out heads and writes only that head's share of qc_out[p] -- its
  // constants, its column of the B-operand fragments with the ones-column beside it, and (h_off == 0) the unused columns.
  constexpr int W = D / 32;
  // G = Hq / Hkv is 1, 2 or 4 (rbq_create): every index split below is a shift or a mask, no integer division
  const int gsh = (Hq >= 4 * Hkv) ? 2 : (Hq >= 2 * Hkv) ? 1 : 0, G = 1 << gsh;
  constexpr int dsh = (D == 64) ? 6 : (D == 128) ? 7 : 8, wsh = dsh - 5;
  if (G_out == 0) G_out = G;                                      // all heads of the group in this call
  const int lane = tid & 31, warp = tid >> 5, nw = nt >> 5;
  auto row0 = [&](int p) { return (size_t)rows0[p]; };             // first query head row (b * Hq + kv head * G) of pair p
  auto sync = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(nt) : "memory"); };

  for (int it = tid; it < NP * G * D; it += nt) {
    const int p = it >> (gsh + dsh), h = (it >> dsh) & (G - 1), j = it & (D - 1);
    const size_t e = (row0(p) + h) * D + j;
    const float qv = rbq_ld_elem(q, e);
    if (q_copy != nullptr) q_copy[e] = q[e];                     // q in mapped host memory: device copy for S7
    const float cqv = c_q ? c_q[e] : 0.0f;
    sm[p].x[h][j] = c_q ? __fsub_rn(qv, cqv) : qv;
    sm[p].y[h][j] = qv;
    sm[p].cq[h][j] = cqv;
    if (h == 0) sm[p].ck[j] = c_k[(size_t)bgs[p] * D + j];
  }
  sync();
  RBQ_QPREP_STAMP(8);
  // ||xq||: the canonical sequential chain, one thread per (pair, head) -- lane 0 of the LAST warps, so that the fp64 dots
  // below (first warps) run beside it
  if (lane == 0 && warp >= nw - NP * G) {
    const int u = warp - (nw - NP * G), p = u >> gsh, h = u & (G - 1);
    float n2 = 0.0f;
#pragma unroll 1
    for (int i0 = 0; i0 < D; i0 += 16) {        // compact loop on purpose: runs once, straight-line code would be fetch-bound
      float4 xv[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) xv[k] = *reinterpret_cast<const float4*>(&sm[p].x[h][i0 + 4 * k]);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        n2 = fmaf(xv[k].x, xv[k].x, n2); n2 = fmaf(xv[k].y, xv[k].y, n2);
        n2 = fmaf(xv[k].z, xv[k].z, n2); n2 = fmaf(xv[k].w, xv[k].w, n2);
      }
    }
    sm[p].qn[h] = __fsqrt_rn(n2);
  }
  // fp64 dots: one warp per (pair, head, 32-dim chunk)
  for (int u = warp; u < NP * G * W; u += nw) {
    const int p = u >> (gsh + wsh), h = (u >> wsh) & (G - 1), w = u & (W - 1), j = 32 * w + lane;
    double p0 = (double)sm[p].y[h][j] * (double)sm[p].ck[j];
    double p1 = c_q ? (double)sm[p].cq[h][j] * (double)sm[p].ck[j] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      p0 += __shfl_xor_sync(0xffffffffu, p0, o);
      p1 += __shfl_xor_sync(0xffffffffu, p1, o);
    }
    if (lane == 0) { sm[p].dred[h][0][w] = p0; sm[p].dred[h][1][w] = p1; }
  }
  sync();
  RBQ_QPREP_STAMP(9);
  for (int it = tid; it < NP * G * D; it += nt) {
    const int p = it >> (gsh + dsh), h = (it >> dsh) & (G - 1), j = it & (D - 1);
    const float qn = sm[p].qn[h];
    sm[p].x[h][j] = (qn > 0.0f) ? __fdiv_rn(sm[p].x[h][j], qn) : 0.0f;
  }
  sync();
  if (rot_kind == RBQ_ROT_DENSE) {
    if (P_SMEM && p_bar_sa != 0u) rbq_mbar_wait(p_bar_sa, 0);
    // one output column for TWO heads of a pair per thread: one read of P[i][j] feeds two independent canonical chains (one
    // read per head is bound by shared-memory bandwidth; all four heads per thread by the issue rate of four lone warps;
    // broadcasting u_i by shuffles instead of 16-byte shared-memory loads was slower still: measured 3.3 K / 3.3 K / 5.7 K clk)
    const int psh = (G > 2) ? 1 : 0, npair = 1 << psh;           // head pairs per KV head: 1 (G = 1, 2) or 2 (G = 4)
    if (G == 1) {
      // one head per pair (single-head mode, or G = 1): one canonical chain per thread; per step one read of P[i][j] and one
      // broadcast of u_i
      for (int it = tid; it < NP * D; it += nt) {
        const int p = it >> dsh, jj = it & (D - 1);
        float a0 = 0.0f;
#pragma unroll 2
        for (int i0 = 0; i0 < D; i0 += 8) {
          float rv[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) rv[k] = P_SMEM ? s_rot[(i0 + k) * D + jj] : __ldg(rot + (size_t)(i0 + k) * D + jj);
          const float4 xa = *reinterpret_cast<const float4*>(&sm[p].x[0][i0]), xb = *reinterpret_cast<const float4*>(&sm[p].x[0][i0 + 4]);
          a0 = fmaf(xa.x, rv[0], a0); a0 = fmaf(xa.y, rv[1], a0); a0 = fmaf(xa.z, rv[2], a0); a0 = fmaf(xa.w, rv[3], a0);
          a0 = fmaf(xb.x, rv[4], a0); a0 = fmaf(xb.y, rv[5], a0); a0 = fmaf(xb.z, rv[6], a0); a0 = fmaf(xb.w, rv[7], a0);
        }
        sm[p].y[0][jj] = a0;
      }
    } else
    for (int it = tid; it < NP * npair * D; it += nt) {
      const int p = it >> (dsh + psh), hp = ((it >> dsh) & (npair - 1)) * 2, jj = it & (D - 1), h1 = min(hp + 1, G - 1);
      float a0 = 0.0f, a1 = 0.0f;
#pragma unroll 2
      for (int i0 = 0; i0 < D; i0 += 8) {
        float rv[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) rv[k] = P_SMEM ? s_rot[(i0 + k) * D + jj] : __ldg(rot + (size_t)(i0 + k) * D + jj);
        const float4 xa = *reinterpret_cast<const float4*>(&sm[p].x[hp][i0]), xb = *reinterpret_cast<const float4*>(&sm[p].x[hp][i0 + 4]);
        const float4 ya = *reinterpret_cast<const float4*>(&sm[p].x[h1][i0]), yb = *reinterpret_cast<const float4*>(&sm[p].x[h1][i0 + 4]);
        a0 = fmaf(xa.x, rv[0], a0); a1 = fmaf(ya.x, rv[0], a1);
        a0 = fmaf(xa.y, rv[1], a0); a1 = fmaf(ya.y, rv[1], a1);
        a0 = fmaf(xa.z, rv[2], a0); a1 = fmaf(ya.z, rv[2], a1);
        a0 = fmaf(xa.w, rv[3], a0); a1 = fmaf(ya.w, rv[3], a1);
        a0 = fmaf(xb.x, rv[4], a0); a1 = fmaf(yb.x, rv[4], a1);
        a0 = fmaf(xb.y, rv[5], a0); a1 = fmaf(yb.y, rv[5], a1);
        a0 = fmaf(xb.z, rv[6], a0); a1 = fmaf(yb.z, rv[6], a1);
        a0 = fmaf(xb.w, rv[7], a0); a1 = fmaf(yb.w, rv[7], a1);
      }
      sm[p].y[hp][jj] = a0;
      if (hp + 1 < G) sm[p].y[hp + 1][jj] = a1;
    }
  } else {
    // Walsh-Hadamard: one warp per (pair, head), W = D/32 consecutive elements per lane; levels h < W in the lane, the
    // others by shuffles (lower lane: a + b, upper lane: a - b with a the lower lane's value)
    for (int uu = warp; uu < NP * G; uu += nw) {
      const int p = uu >> gsh, h = uu & (G - 1);
      float u[W];
#pragma unroll
      for (int e = 0; e < W; ++e) u[e] = __fmul_rn(rot[lane * W + e], sm[p].x[h][lane * W + e]);
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
      for (int m = 1; m < 32; m <<= 1) {
        const bool up = (lane & m) != 0;
#pragma unroll
        for (int e = 0; e < W; ++e) {
          const float pp = __shfl_xor_sync(0xffffffffu, u[e], m);
          u[e] = up ? __fsub_rn(pp, u[e]) : __fadd_rn(u[e], pp);
        }
      }
      const float c1 = (float)(1.0 / sqrt((double)D));
#pragma unroll
      for (int e = 0; e < W; ++e) sm[p].y[h][lane * W + e] = __fmul_rn(u[e], c1);
    }
  }
  sync();
  RBQ_QPREP_STAMP(10);
  // one warp per (pair, head, 32-dim chunk): min / max over ALL D rotated coordinates of the head (every chunk warp reduces
  // the whole row: W values per lane + a shuffle tree), Delta, the INT4 codes of its chunk and their sum
  for (int uu = warp; uu < NP * G * W; uu += nw) {
    const int p = uu >> (gsh + wsh), h = (uu >> wsh) & (G - 1), w = uu & (W - 1);
    float v[W];
#pragma unroll
    for (int e = 0; e < W; ++e) v[e] = sm[p].y[h][32 * e + lane];
    float ql = v[0], qr = v[0], mine = v[0];
#pragma unroll
    for (int e = 1; e < W; ++e) { ql = fminf(ql, v[e]); qr = fmaxf(qr, v[e]); mine = (e == w) ? v[e] : mine; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      ql = fminf(ql, __shfl_xor_sync(0xffffffffu, ql, o));
      qr = fmaxf(qr, __shfl_xor_sync(0xffffffffu, qr, o));
    }
    const float delta = __fdiv_rn(__fsub_rn(qr, ql), 15.0f);
    int c = 0;
    if (delta > 0.0f) {
      const float t = __fdiv_rn(__fsub_rn(mine, ql), delta);
      c = (int)floorf(__fadd_rn(t, 0.5f));
      c = min(15, max(0, c));
    }
    sm[p].qu[h][32 * w + lane] = (uint8_t)c;
    if (qu_out) qu_out[(row0(p) + h) * D + 32 * w + lane] = (uint8_t)c;
    int sv = c;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sv += __shfl_xor_sync(0xffffffffu, sv, o);
    if (lane == 0) {
      sm[p].isum[h][w] = sv;
      if (w == 0) { sm[p].ql[h] = ql; sm[p].delta[h] = delta; }
    }
  }
  sync();
  // the Eq.20 / Eq.2 constants: one thread per (pair, head)
  if (tid < NP * G) {
    const int p = tid >> gsh, h = tid & (G - 1);
    int sumq = 0;
    double d0[W], d1[W];
#pragma unroll
    for (int k = 0; k < W; ++k) { sumq += sm[p].isum[h][k]; d0[k] = sm[p].dred[h][0][k]; d1[k] = sm[p].dred[h][1][k]; }
#pragma unroll
    for (int st = 1; st < W; st <<= 1) {          // pairwise tree: (d0 + d1) + (d2 + d3) ...
#pragma unroll
      for (int k = 0; k < W; k += 2 * st) { d0[k] += d0[k + st]; d1[k] += d1[k + st]; }
    }
    const float ql = sm[p].ql[h], delta = sm[p].delta[h];
    const float qn = sm[p].qn[h], q_ck = (float)d0[0], cq_ck = (float)d1[0];
    if (qparams) {
      float* o = qparams + (row0(p) + h) * 6;
      o[0] = qn; o[1] = ql; o[2] = delta; o[3] = (float)sumq; o[4] = q_ck; o[5] = cq_ck;
    }
    const int ho = h + h_off;
    qc_out[p].cA[ho] = (float)((double)sm_scale * (double)qn * (double)delta * 0.25);
    qc_out[p].cB[ho] = (float)((double)sm_scale * (double)qn * (double)ql * 0.25);
    qc_out[p].cD[ho] = (float)((double)sm_scale * ((double)q_ck - (double)cq_ck));
    qc_out[p].init_d[ho] = 0x4B400000 - 4 * sumq;
    if (ho == 0) qc_out[p].init_p = 0x4B400000 - 4 * D;
  }
  RBQ_QPREP_STAMP(14);
  // B-operand fragments (rbq_bfrag_dim): word (s, lane', r), byte i; column n = lane' >> 2: even -> head n/2, odd -> ones
  for (int w0 = tid; w0 < NP * W * 64; w0 += nt) {
    const int p = w0 >> (wsh + 6), w = w0 & (W * 64 - 1);
    const int s = w >> 6, ln = (w >> 1) & 31, r = w & 1;
    const int gp = ln >> 2, tp = ln & 3, hc = gp >> 1;             // hc: the head this column (or its ones-column) belongs to
    const bool mine = (hc >= h_off && hc < h_off + G) || (h_off == 0 && hc >= G_out);
    if (!mine) continue;
    uint32_t word = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      int dim, sh;
      rbq_bfrag_dim(W, s, tp, r, i, dim, sh);
      uint32_t val = 0;
      if (gp & 1) val = (hc < G_out) ? 1u : 0u;
      else if (hc < G_out) val = sm[p].qu[hc - h_off][dim];
      word |= (val << sh) << (8 * i);
    }
    qc_out[p].bfrag[s][ln][r] = word;
  }
}
