/*
 * rbq_ref.c -- CPU ORACLE for the RaBitQCache decode hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code with paper_2606_31519_b200/csrc (the CUDA path) and neither
 * side includes or imports the other.
 *
 * Plain, slow, single-file C written from /root/reference/PAPER.md
 * (arxiv/paper_2606_31519).  Every function cites the passage it follows
 * ("PAPER.md:L<n>").  Readings of silent/garbled passages are the ones listed in
 * DESIGN.md section 3 ("Readings") and are referred to here as R1..R16.
 *
 * Precision policy
 *   - Steps whose result is an INTEGER decision that the GPU must reproduce
 *     bit-for-bit (sign bits of the rotated key, INT4 query codes) and the
 *     stored fp32 factors are computed in a CANONICAL FP32 ORDER (R1): IEEE
 *     binary32, round-to-nearest-even, explicit fmaf(), ascending index, one
 *     accumulator per output, no reassociation.  Compile with
 *     -ffp-contract=off and WITHOUT -ffast-math.
 *   - Everything else (logits from stored values, softmax, Top-p, attention)
 *     is fp64.
 *
 * Parity pins (tests/test_oracle_*.py): rotation orthogonality and agreement
 * with numpy QR; packed == unpacked integer dot; Eq.20 == direct <c', q_bar>;
 * Eq.2 identity; unbiasedness law of Thm A.1 / Lemma A.4 and the closed form
 * of E[alpha]; encode invariants; Top-p minimality vs brute force over subsets
 * and vs Alg.3; p=1 == dense softmax attention (numpy); worked literal config.
 * The paper prints no worked numeric example of codes/alpha/scores, so absolute
 * agreement with the authors' implementation is "parity unpinned".
 *
 * Layouts: all arrays are host memory, contiguous, row-major; K and V are
 * float32 [B][Hkv][Lcap][D] (bf16 inputs are widened exactly by the caller).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define RBQ_REF_OK 0
#define RBQ_REF_ERR (-1)

enum { RBQ_REF_ROT_DENSE = 0, RBQ_REF_ROT_WH = 1 };

/* ------------------------------------------------------------------------- */
/* threads                                                                    */
/* ------------------------------------------------------------------------- */
int rbq_ref_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void rbq_ref_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ------------------------------------------------------------------------- */
/* O1  random orthogonal rotation P  ("random orthogonal rotation  */
/*     matrix P", L149 "generated once during model initialization", L567       */
/*     "drawn uniformly from the Haar measure").                                */
/*     Householder QR of a Gaussian matrix A = Q*Rt in fp64, then               */
/*     Q*diag(sign(diag(Rt))) (the unique factor with positive diagonal, which   */
/*     is Haar distributed), rounded to fp32.  rot[i][j] row-major.             */
/* ------------------------------------------------------------------------- */
int rbq_ref_rotation_from_gaussian(const double* A, int D, float* rot32, double* rot64) {
  if (!A || D <= 0 || !rot32) return RBQ_REF_ERR;
  double* M = (double*)malloc(sizeof(double) * D * D); /* becomes Rt */
  double* Q = (double*)malloc(sizeof(double) * D * D);
  double* v = (double*)malloc(sizeof(double) * D);
  if (!M || !Q || !v) { free(M); free(Q); free(v); return RBQ_REF_ERR; }
  memcpy(M, A, sizeof(double) * D * D);
  for (int i = 0; i < D; ++i)
    for (int j = 0; j < D; ++j) Q[i * D + j] = (i == j) ? 1.0 : 0.0;
  for (int k = 0; k < D; ++k) {
    /* Householder vector for column k, rows k..D-1 */
    double nrm = 0.0;
    for (int i = k; i < D; ++i) nrm += M[i * D + k] * M[i * D + k];
    nrm = sqrt(nrm);
    if (nrm == 0.0) continue;
    double a = M[k * D + k];
    double beta = (a >= 0.0) ? -nrm : nrm; /* reflect x onto beta*e_k */
    for (int i = 0; i < D; ++i) v[i] = 0.0;
    v[k] = a - beta;
    for (int i = k + 1; i < D; ++i) v[i] = M[i * D + k];
    double vv = 0.0;
    for (int i = k; i < D; ++i) vv += v[i] * v[i];
    if (vv == 0.0) continue;
    /* M <- (I - 2 v v^T / vv) M ;  Q <- Q (I - 2 v v^T / vv) */
    for (int j = 0; j < D; ++j) {
      double s = 0.0;
      for (int i = k; i < D; ++i) s += v[i] * M[i * D + j];
      s = 2.0 * s / vv;
      for (int i = k; i < D; ++i) M[i * D + j] -= s * v[i];
    }
    for (int i = 0; i < D; ++i) {
      double s = 0.0;
      for (int j = k; j < D; ++j) s += Q[i * D + j] * v[j];
      s = 2.0 * s / vv;
      for (int j = k; j < D; ++j) Q[i * D + j] -= s * v[j];
    }
  }
  for (int j = 0; j < D; ++j) {
    double sgn = (M[j * D + j] < 0.0) ? -1.0 : 1.0;
    for (int i = 0; i < D; ++i) {
      double q = Q[i * D + j] * sgn;
      if (rot64) rot64[i * D + j] = q;
      rot32[i * D + j] = (float)q;
    }
  }
  free(M); free(Q); free(v);
  return RBQ_REF_OK;
}

/* Unscaled in-place fast Walsh-Hadamard transform, Sylvester ordering.       */
/* Canonical butterfly order (R1): h = 1,2,4,...,D/2; (a,b) -> (a+b, a-b).     */
/* Not in the paper (it only cites FJLT); the WH rotation is     */
/* BASELINE.json config 4's addition.                                          */
static void fwht_f32(float* u, int D) {
  for (int h = 1; h < D; h <<= 1)
    for (int i = 0; i < D; i += (h << 1))
      for (int j = i; j < i + h; ++j) {
        float a = u[j], b = u[j + h];
        u[j] = a + b;
        u[j + h] = a - b;
      }
}
void rbq_ref_fwht(float* u, int D) { fwht_f32(u, D); }

/* Materialised WH rotation: rot[i][j] = s_i * H[i][j] / sqrt(D), H Sylvester  */
/* (H[i][j] = (-1)^popcount(i&j)); y = x * rot  ==  H (s .* x) / sqrt(D).      */
int rbq_ref_rotation_wh(const float* s, int D, float* rot32) {
  if (!s || !rot32 || D <= 0 || (D & (D - 1))) return RBQ_REF_ERR;
  double inv = 1.0 / sqrt((double)D);
  for (int i = 0; i < D; ++i)
    for (int j = 0; j < D; ++j) {
      int par = __builtin_popcount((unsigned)(i & j)) & 1;
      rot32[i * D + j] = (float)((par ? -1.0 : 1.0) * (double)s[i] * inv);
    }
  return RBQ_REF_OK;
}

/* y = x * rot in the canonical fp32 order (R1).                              */
/*  DENSE: y_j = fma-chain over i ascending of x_i*rot[i][j], acc starts at 0. */
/*  WH   : u = s.*x ; butterflies ; y_j = u_j * fl32(1/sqrt(D)).               */
/*         `y_unscaled` (may be NULL) receives u after the butterflies.        */
static void rotate_canonical(const float* x, int D, int rot_kind, const float* rot, float* y,
                             float* y_unscaled) {
  if (rot_kind == RBQ_REF_ROT_DENSE) {
    for (int j = 0; j < D; ++j) y[j] = 0.0f;
    for (int i = 0; i < D; ++i) {
      const float xi = x[i];
      const float* r = rot + (size_t)i * D;
      for (int j = 0; j < D; ++j) y[j] = fmaf(xi, r[j], y[j]);
    }
    if (y_unscaled) memcpy(y_unscaled, y, sizeof(float) * D);
  } else {
    const float c = (float)(1.0 / sqrt((double)D));
    for (int i = 0; i < D; ++i) y[i] = rot[i] * x[i]; /* s_i in {-1,+1}: exact */
    fwht_f32(y, D);
    if (y_unscaled) memcpy(y_unscaled, y, sizeof(float) * D);
    for (int j = 0; j < D; ++j) y[j] = y[j] * c;
  }
}

/* ------------------------------------------------------------------------- */
/* O2a centroid c_k = mean of the prefill keys ("Calculate        */
/*     centroid c_k from K", L66 "centroids of the prefilling ... key vectors").*/
/*     fp64 sum over t ascending, divided by n, rounded to fp32.               */
/* ------------------------------------------------------------------------- */
int rbq_ref_centroid(const float* K, int B, int Hkv, int Lcap, int D, const int32_t* seq_lens,
                     float* c_k) {
  if (!K || !seq_lens || !c_k) return RBQ_REF_ERR;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hkv; ++h) {
      const float* Kh = K + ((size_t)b * Hkv + h) * Lcap * D;
      int n = seq_lens[b];
      for (int d = 0; d < D; ++d) {
        double s = 0.0;
        for (int t = 0; t < n; ++t) s += (double)Kh[(size_t)t * D + d];
        c_k[((size_t)b * Hkv + h) * D + d] = (n > 0) ? (float)(s / (double)n) : 0.0f;
      }
    }
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O2b Alg.1 index construction (L149-151; L485-487).        */
/*   for tokens t in [t_begin[b], t_end[b]) of every (b, kv head):             */
/*     x  = k_t - c_k                      (Alg.1 line 6, fp32 subtraction)    */
/*     n2 = ||x||^2                        (fma chain, i ascending)            */
/*     y  = x * P                          (Alg.1 line 10 / L149, R2: y_j =     */
/*                                          sum_i x_i P[i][j] = (P^T x)_j)     */
/*     bit_j = [y_j > 0]                   (L485: "1 if ... positive, 0 otherwise")*/
/*     codes: dim j -> word j/32, bit j%32 (L270 "pack 32 consecutive binary   */
/*                                          elements ... into a 32-bit integer", R10) */
/*     l1 = ||y||_1                        (sequential sum, j ascending)       */
/*     f_scale = n2 / l1  (0 if l1 == 0)   (R4: = ||k-c_k|| / <c', P^T k_c>,   */
/*        because <c', P^T k_c> = ||y||_1/||x||_2 -- Eq.18; the      */
/*        sign pattern is scale invariant so the un-normalised x is rotated,   */
/*        R3)                                                                  */
/*     f_bias[b][hq][t] = <c_q[b][hq], k_t> (L89 "<c_q,k> ... can be            */
/*        pre-calculated"), fma chain i ascending; only when c_q != NULL.      */
/* ------------------------------------------------------------------------- */
int rbq_ref_encode(const float* K, int B, int Hkv, int Lcap, int D, const int32_t* t_begin,
                   const int32_t* t_end, int rot_kind, const float* rot, const float* c_k,
                   const float* c_q, int Hq, uint32_t* codes, float* f_scale, float* f_bias) {
  if (!K || !t_begin || !t_end || !rot || !c_k || !codes || !f_scale) return RBQ_REF_ERR;
  if (D % 32 != 0 || D > 1024) return RBQ_REF_ERR;
  if (c_q && (!f_bias || Hq % Hkv != 0)) return RBQ_REF_ERR;
  const int W = D / 32;
  const int G = c_q ? Hq / Hkv : 0;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hkv; ++h) {
      const float* Kh = K + ((size_t)b * Hkv + h) * Lcap * D;
      const float* ck = c_k + ((size_t)b * Hkv + h) * D;
      uint32_t* ch = codes + ((size_t)b * Hkv + h) * Lcap * W;
      float* fh = f_scale + ((size_t)b * Hkv + h) * Lcap;
      int t0 = t_begin[b], t1 = t_end[b];
#pragma omp parallel for schedule(static)
      for (int t = t0; t < t1; ++t) {
        float x[1024], y[1024];
        const float* k = Kh + (size_t)t * D;
        for (int i = 0; i < D; ++i) x[i] = k[i] - ck[i];
        float n2 = 0.0f;
        for (int i = 0; i < D; ++i) n2 = fmaf(x[i], x[i], n2);
        float yu[1024];
        rotate_canonical(x, D, rot_kind, rot, y, yu);
        float l1 = 0.0f;
        if (rot_kind == RBQ_REF_ROT_DENSE) {
          for (int j = 0; j < D; ++j) l1 = l1 + fabsf(y[j]);
        } else { /* WH: ||y||_1 = (sum_j |u_j|, j ascending) * fl32(1/sqrt(D))  (R1) */
          for (int j = 0; j < D; ++j) l1 = l1 + fabsf(yu[j]);
          l1 = l1 * (float)(1.0 / sqrt((double)D));
        }
        for (int w = 0; w < W; ++w) {
          uint32_t word = 0;
          for (int j = 0; j < 32; ++j)
            if (y[w * 32 + j] > 0.0f) word |= (1u << j);
          ch[(size_t)t * W + w] = word;
        }
        fh[t] = (l1 == 0.0f) ? 0.0f : n2 / l1;
        for (int g = 0; g < G; ++g) {
          int hq = h * G + g;
          const float* cq = c_q + ((size_t)b * Hq + hq) * D;
          float acc = 0.0f;
          for (int i = 0; i < D; ++i) acc = fmaf(cq[i], k[i], acc);
          f_bias[((size_t)b * Hq + hq) * Lcap + t] = acc;
        }
      }
    }
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O2c 2-byte correction factors ("B_alpha ... typically FP16",   */
/*     L756-766: the 3.5 % space figure assumes an FP16 factor per token and    */
/*     head).  The stored factor f_scale (R4) is rounded to IEEE binary16,      */
/*     round-to-nearest-even, and widened back: every later step (O5) then      */
/*     uses the rounded value exactly as it uses the fp32 one.  Overflow to inf */
/*     cannot happen for finite keys of the workloads (f_scale ~ ||x||/sqrt(D)); */
/*     values below the binary16 subnormal range round to 0 (the estimated part */
/*     of such a logit is then dropped, as for x = 0, R15).                     */
/* ------------------------------------------------------------------------- */
int rbq_ref_round_factors_f16(float* f_scale, long long n) {
  if (!f_scale || n < 0) return RBQ_REF_ERR;
  for (long long i = 0; i < n; ++i) f_scale[i] = (float)(_Float16)f_scale[i];
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O3  query pre-processing and INT4 quantisation                              */
/*     (Alg.2 lines 4-6; L192-197 Eq.5; L524).               */
/*   xq = q - c_q ; qn = ||xq||_2 ; u = xq/qn      (Alg.2 line 4, R12)         */
/*   q' = u * P                                    (Alg.2 line 5, same P, R2)  */
/*   q_l = min q', q_r = max q', Delta = (q_r-q_l)/(2^4-1)   (L524, R5)        */
/*   qu_j = clamp(floor((q'_j - q_l)/Delta + 1/2), 0, 15)    (Eq.5, R6)        */
/*   all in the canonical fp32 order (the INT4 codes are an integer decision   */
/*   that both sides take in fp32).  Delta == 0 -> qu = 0 (R5).                */
/*   Per (b,hq) scalars also returned: sumq = sum qu ;                         */
/*   q_ck = <q, c_k>, cq_ck = <c_q, c_k> (fp64 -> fp32; Eq.2 L86 terms).       */
/* ------------------------------------------------------------------------- */
int rbq_ref_query_prep(const float* q, int B, int Hq, int Hkv, int D, int rot_kind,
                       const float* rot, const float* c_q, const float* c_k, uint8_t* qu,
                       float* qn_out, float* ql_out, float* delta_out, int32_t* sumq_out,
                       float* q_ck_out, float* cq_ck_out, float* qprime_out) {
  if (!q || !rot || !c_k || !qu || !qn_out || !ql_out || !delta_out || !sumq_out || !q_ck_out ||
      !cq_ck_out)
    return RBQ_REF_ERR;
  if (D > 1024 || Hq % Hkv != 0) return RBQ_REF_ERR;
  const int G = Hq / Hkv;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hq; ++h) {
      const size_t r = (size_t)b * Hq + h;
      const float* qv = q + r * D;
      const float* cq = c_q ? c_q + r * D : NULL;
      const float* ck = c_k + ((size_t)b * Hkv + h / G) * D;
      float xq[1024], u[1024], qp[1024];
      for (int i = 0; i < D; ++i) xq[i] = cq ? (qv[i] - cq[i]) : qv[i];
      float n2 = 0.0f;
      for (int i = 0; i < D; ++i) n2 = fmaf(xq[i], xq[i], n2);
      float qn = sqrtf(n2);
      for (int i = 0; i < D; ++i) u[i] = (qn > 0.0f) ? xq[i] / qn : 0.0f;
      rotate_canonical(u, D, rot_kind, rot, qp, NULL);
      float ql = qp[0], qr = qp[0];
      for (int j = 1; j < D; ++j) {
        if (qp[j] < ql) ql = qp[j];
        if (qp[j] > qr) qr = qp[j];
      }
      float delta = (qr - ql) / 15.0f;
      int32_t sumq = 0;
      for (int j = 0; j < D; ++j) {
        int v = 0;
        if (delta > 0.0f) {
          float t = (qp[j] - ql) / delta;
          float fl = floorf(t + 0.5f);
          v = (int)fl;
          if (v < 0) v = 0;
          if (v > 15) v = 15;
        }
        qu[r * D + j] = (uint8_t)v;
        sumq += v;
      }
      double a = 0.0, c = 0.0;
      for (int i = 0; i < D; ++i) {
        a += (double)qv[i] * (double)ck[i];
        if (cq) c += (double)cq[i] * (double)ck[i];
      }
      qn_out[r] = qn;
      ql_out[r] = ql;
      delta_out[r] = delta;
      sumq_out[r] = sumq;
      q_ck_out[r] = (float)a;
      cq_ck_out[r] = (float)c;
      if (qprime_out) memcpy(qprime_out + r * D, qp, sizeof(float) * D);
    }
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O4  Int4_Dot_Binary (Alg.2 line 8; L268-274; L534):           */
/*     dot[b][hq][t] = <c_b[t], qu> = sum_j bit_{t,j} * qu_j,                   */
/*     pop[b][hkv][t] = sum_j bit_{t,j}, for t < n_indexed[b].                 */
/*     (a) brute force over the UNPACKED vectors; (b) packed bit-plane form    */
/*     sum_{p=0..3} 2^p popcount(word & plane_p(qu)).  (a) is the definition;  */
/*     tests require (a) == (b) exactly.                                       */
/* ------------------------------------------------------------------------- */
int rbq_ref_int_dots(const uint32_t* codes, const uint8_t* qu, int B, int Hq, int Hkv, int Lcap,
                     int D, const int32_t* n_indexed, int32_t* dot, int32_t* pop) {
  if (!codes || !qu || !n_indexed || !dot || !pop || D % 32 || Hq % Hkv) return RBQ_REF_ERR;
  const int W = D / 32, G = Hq / Hkv;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hq; ++h) {
      const uint32_t* ch = codes + ((size_t)b * Hkv + h / G) * Lcap * W;
      const uint8_t* quv = qu + ((size_t)b * Hq + h) * D;
      int32_t* dh = dot + ((size_t)b * Hq + h) * Lcap;
      int32_t* ph = pop + ((size_t)b * Hkv + h / G) * Lcap;
      int n = n_indexed[b];
#pragma omp parallel for schedule(static)
      for (int t = 0; t < n; ++t) {
        int32_t s = 0, c = 0;
        for (int j = 0; j < D; ++j) {
          int bit = (int)((ch[(size_t)t * W + j / 32] >> (j % 32)) & 1u);
          s += bit * (int)quv[j];
          c += bit;
        }
        dh[t] = s;
        if (h % G == 0) ph[t] = c;
      }
    }
  return RBQ_REF_OK;
}

int rbq_ref_int_dots_packed(const uint32_t* codes, const uint8_t* qu, int B, int Hq, int Hkv,
                            int Lcap, int D, const int32_t* n_indexed, int32_t* dot,
                            int32_t* pop) {
  if (!codes || !qu || !n_indexed || !dot || !pop || D % 32 || D > 1024 || Hq % Hkv)
    return RBQ_REF_ERR;
  const int W = D / 32, G = Hq / Hkv;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hq; ++h) {
      const uint32_t* ch = codes + ((size_t)b * Hkv + h / G) * Lcap * W;
      const uint8_t* quv = qu + ((size_t)b * Hq + h) * D;
      uint32_t plane[4][32];
      for (int p = 0; p < 4; ++p)
        for (int w = 0; w < W; ++w) {
          uint32_t m = 0;
          for (int j = 0; j < 32; ++j) m |= (uint32_t)((quv[w * 32 + j] >> p) & 1u) << j;
          plane[p][w] = m;
        }
      int32_t* dh = dot + ((size_t)b * Hq + h) * Lcap;
      int32_t* ph = pop + ((size_t)b * Hkv + h / G) * Lcap;
      int n = n_indexed[b];
      for (int t = 0; t < n; ++t) {
        int32_t s = 0, c = 0;
        for (int w = 0; w < W; ++w) {
          uint32_t cw = ch[(size_t)t * W + w];
          for (int p = 0; p < 4; ++p) s += __builtin_popcount(cw & plane[p][w]) << p;
          c += __builtin_popcount(cw);
        }
        dh[t] = s;
        if (h % G == 0) ph[t] = c;
      }
    }
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O5  Reconstruct + Eq.2 (Alg.2 lines 9-10; Eq.20;      */
/*     Eq.18; Eq.2; softmax scale L184):                              */
/*   ip    = 2*Delta*dot + 2*q_l*pop - Delta*sumq - D*q_l      (Eq.20)         */
/*   S     = qn * f_scale * ip + <q,c_k> + f_bias - <c_q,c_k>  (Eq.18 + Eq.2)  */
/*   score = S * sm_scale                                      (L184, R11)     */
/*   in fp64 from the stored fp32 values, rounded to fp32 once.               */
/* ------------------------------------------------------------------------- */
int rbq_ref_logits(const int32_t* dot, const int32_t* pop, const float* f_scale,
                   const float* f_bias, const float* qn, const float* ql, const float* delta,
                   const int32_t* sumq, const float* q_ck, const float* cq_ck, int B, int Hq,
                   int Hkv, int Lcap, int D, const int32_t* n_indexed, double sm_scale,
                   float* scores) {
  if (!dot || !pop || !f_scale || !qn || !ql || !delta || !sumq || !q_ck || !cq_ck || !scores ||
      Hq % Hkv)
    return RBQ_REF_ERR;
  const int G = Hq / Hkv;
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hq; ++h) {
      const size_t r = (size_t)b * Hq + h;
      const int32_t* dh = dot + r * Lcap;
      const int32_t* ph = pop + ((size_t)b * Hkv + h / G) * Lcap;
      const float* fs = f_scale + ((size_t)b * Hkv + h / G) * Lcap;
      const float* fb = f_bias ? f_bias + r * Lcap : NULL;
      const double dl = (double)delta[r], l = (double)ql[r], n = (double)qn[r];
      const double cst = (double)q_ck[r] - (double)cq_ck[r];
      int nidx = n_indexed[b];
      for (int t = 0; t < nidx; ++t) {
        double ip = 2.0 * dl * (double)dh[t] + 2.0 * l * (double)ph[t] - dl * (double)sumq[r] -
                    (double)D * l;
        double S = n * (double)fs[t] * ip + cst + (fb ? (double)fb[t] : 0.0);
        scores[r * Lcap + t] = (float)(S * sm_scale);
      }
    }
  return RBQ_REF_OK;
}

/* ------------------------------------------------------------------------- */
/* O6  Adaptive Top-p selection (Alg.2 line 12; L201 "the minimum */
/*     set of indices I_select required to cover the probability mass p").     */
/*   per row of n scores: m = max; w_t = exp(score_t - m) (fp64); Z = sum w;   */
/*   order by (w desc, t asc) (R8: lowest index wins ties); I = shortest       */
/*   prefix with cumulative w >= p*Z.  p >= 1 -> all n (R9).  n = 0 -> empty.  */
/*   sel_idx row receives I in that order; sel_cnt its size.                   */
/* ------------------------------------------------------------------------- */
typedef struct { double w; int32_t t; } wt_pair;
static int cmp_wt(const void* a, const void* b) {
  const wt_pair* x = (const wt_pair*)a; const wt_pair* y = (const wt_pair*)b;
  if (x->w > y->w) return -1;
  if (x->w < y->w) return 1;
  return (x->t < y->t) ? -1 : (x->t > y->t);
}
int rbq_ref_topp(const float* scores, int rows, int Lcap, const int32_t* n_per_row, double p,
                 int32_t* sel_idx, int32_t* sel_cnt) {
  if (!scores || !n_per_row || !sel_idx || !sel_cnt) return RBQ_REF_ERR;
  int err = 0;
#pragma omp parallel for schedule(dynamic)
  for (int r = 0; r < rows; ++r) {
    const float* s = scores + (size_t)r * Lcap;
    int32_t* out = sel_idx + (size_t)r * Lcap;
    int n = n_per_row[r];
    if (n <= 0) { sel_cnt[r] = 0; continue; }
    if (p >= 1.0) {
      for (int t = 0; t < n; ++t) out[t] = t;
      sel_cnt[r] = n;
      continue;
    }
    wt_pair* a = (wt_pair*)malloc(sizeof(wt_pair) * (size_t)n);
    if (!a) { err = 1; continue; }
    double m = (double)s[0];
    for (int t = 1; t < n; ++t) if ((double)s[t] > m) m = (double)s[t];
    double Z = 0.0;
    for (int t = 0; t < n; ++t) { a[t].w = exp((double)s[t] - m); a[t].t = t; Z += a[t].w; }
    qsort(a, (size_t)n, sizeof(wt_pair), cmp_wt);
    double cum = 0.0, target = p * Z;
    int k = 0;
    while (k < n && cum < target) { cum += a[k].w; ++k; }
    for (int i = 0; i < k; ++i) out[i] = a[i].t;
    sel_cnt[r] = k;
    free(a);
  }
  return err ? RBQ_REF_ERR : RBQ_REF_OK;
}

/* Alg.3 "Top-p Mask Generation Logic" on one row of       */
/* probabilities prob[0..n) (sum 1).  The listing lost an `else` between L242  */
/* and L245; restored per the text at L262-264 (R13):                          */
/*   low<-0, high<-max S; repeat { pi0=(high+2low)/3; pi1=(2high+low)/3;       */
/*   G0=sum s[s>pi0]; G1=sum s[s>pi1]; vmin=min{s>low}; vmax=max{s<=high};     */
/*   if G1>=p: low<-pi1  elif G0>=p: low<-pi0, high<-min(pi1,vmax)             */
/*   else: high<-min(pi0,vmax) } until vmin==vmax; theta<-low; M<-(S>theta).   */
/* Cross-check only: its mask must equal {t : w_t >= w_(k)} which contains     */
/* the minimal set of rbq_ref_topp and equals it when the boundary value is    */
/* unique.  Returns the iteration count, or -1.                                */
int rbq_ref_topp_alg3(const double* prob, int n, double p, uint8_t* mask) {
  if (!prob || !mask || n <= 0) return -1;
  double low = 0.0, high = prob[0];
  for (int t = 1; t < n; ++t) if (prob[t] > high) high = prob[t];
  int it = 0;
  for (;;) {
    ++it;
    double pi0 = (high + 2.0 * low) / 3.0, pi1 = (2.0 * high + low) / 3.0;
    double G0 = 0.0, G1 = 0.0, vmin = INFINITY, vmax = -INFINITY;
    for (int t = 0; t < n; ++t) {
      double s = prob[t];
      if (s > pi0) G0 += s;
      if (s > pi1) G1 += s;
      if (s > low && s < vmin) vmin = s;
      if (s <= high && s > vmax) vmax = s;
    }
    if (G1 >= p) low = pi1;
    else if (G0 >= p) { low = pi0; high = (pi1 < vmax) ? pi1 : vmax; }
    else high = (pi0 < vmax) ? pi0 : vmax;
    if (vmin == vmax || it > 4096) break;
  }
  for (int t = 0; t < n; ++t) mask[t] = (prob[t] > low) ? 1 : 0;
  return it;
}

/* ------------------------------------------------------------------------- */
/* O7  Hybrid attention over the selected tokens and the local window          */
/*     (Alg.2 lines 14-15; L215 "K_local acts as a           */
/*     full-precision write-back buffer ... participate in the hybrid          */
/*     attention").  A = sel_idx[b][h][0..cnt) U [n_indexed[b], n_total[b]);   */
/*     l_t = <q,k_t>*sm_scale; o = sum_A softmax_A(l)_t v_t (renormalised over */
/*     A, R7); lse = log sum_A exp(l_t).  fp64, rounded to fp32 at the end.    */
/*     Empty A -> o = 0, lse = -inf.                                           */
/* ------------------------------------------------------------------------- */
int rbq_ref_attention(const float* q, const float* K, const float* V, int B, int Hq, int Hkv,
                      int Lcap, int D, const int32_t* sel_idx, const int32_t* sel_cnt,
                      const int32_t* n_indexed, const int32_t* n_total, double sm_scale,
                      float* out, float* lse) {
  if (!q || !K || !V || !sel_idx || !sel_cnt || !n_indexed || !n_total || !out || Hq % Hkv)
    return RBQ_REF_ERR;
  const int G = Hq / Hkv;
  int err = 0;
#pragma omp parallel for collapse(2) schedule(dynamic)
  for (int b = 0; b < B; ++b)
    for (int h = 0; h < Hq; ++h) {
      const size_t r = (size_t)b * Hq + h;
      const float* qv = q + r * D;
      const float* Kh = K + ((size_t)b * Hkv + h / G) * Lcap * D;
      const float* Vh = V + ((size_t)b * Hkv + h / G) * Lcap * D;
      const int32_t* idx = sel_idx + r * Lcap;
      int cnt = sel_cnt[r];
      int npend = n_total[b] - n_indexed[b];
      int na = cnt + (npend > 0 ? npend : 0);
      float* o = out + r * D;
      if (na == 0) {
        for (int d = 0; d < D; ++d) o[d] = 0.0f;
        if (lse) lse[r] = -INFINITY;
        continue;
      }
      double* l = (double*)malloc(sizeof(double) * (size_t)na);
      int32_t* tok = (int32_t*)malloc(sizeof(int32_t) * (size_t)na);
      double* acc = (double*)calloc((size_t)D, sizeof(double));
      if (!l || !tok || !acc) { err = 1; free(l); free(tok); free(acc); continue; }
      for (int i = 0; i < cnt; ++i) tok[i] = idx[i];
      for (int i = cnt; i < na; ++i) tok[i] = n_indexed[b] + (i - cnt);
      double m = -INFINITY;
      for (int i = 0; i < na; ++i) {
        const float* k = Kh + (size_t)tok[i] * D;
        double s = 0.0;
        for (int d = 0; d < D; ++d) s += (double)qv[d] * (double)k[d];
        l[i] = s * sm_scale;
        if (l[i] > m) m = l[i];
      }
      double Z = 0.0;
      for (int i = 0; i < na; ++i) {
        double w = exp(l[i] - m);
        Z += w;
        const float* v = Vh + (size_t)tok[i] * D;
        for (int d = 0; d < D; ++d) acc[d] += w * (double)v[d];
      }
      for (int d = 0; d < D; ++d) o[d] = (float)(acc[d] / Z);
      if (lse) lse[r] = (float)(m + log(Z));
      free(l); free(tok); free(acc);
    }
  return err ? RBQ_REF_ERR : RBQ_REF_OK;
}
