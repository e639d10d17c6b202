"""Pins for oracle O3-O5 (query INT4, binary x INT4 dot, reconstruction, Eq.2).  CPU only.

P2  packed bit-plane dot == brute-force integer dot of the unpacked vectors == numpy matmul.
P7  Eq.20 == <2c_b-1, Delta*qu+q_l> evaluated directly; Eq.2 (L86) is an
    identity for any c_q, c_k when the exact cosine is plugged in.
P3  unbiasedness law of Thm A.1 / Lemma A.4 (L509-514, L567-572, density L558) over seeded
    Haar rotations; P4 closed form E[alpha] = sqrt(D) Gamma(D/2) / (sqrt(pi) Gamma((D+1)/2)).
O3  INT4 quantiser (Eq.5): range, clamp, reconstruction error <= Delta/2.
"""
import math
from pathlib import Path

import numpy as np
import pytest
from scipy.special import gammaln

from paper_2606_31519_b200 import synth
from tests.test_oracle_rotation_encode import unpack

D = 128
GOLD = Path(__file__).parent / "golden"


def _planes_dot_numpy(codes, qu):
    bits = unpack(codes)                       # [..., L, D]
    return bits @ qu.astype(np.int64)


def test_p2_packed_equals_bruteforce_equals_numpy(orc):
    rng = np.random.default_rng(2)
    B, Hq, Hkv, L = 2, 8, 2, 300
    codes = rng.integers(0, 2 ** 32, (B, Hkv, L, 4), dtype=np.uint64).astype(np.uint32)
    # adversarial codes
    codes[0, 0, 0] = 0
    codes[0, 0, 1] = 0xFFFFFFFF
    codes[0, 0, 2] = [1, 0, 0, 0]
    codes[0, 0, 3] = [0, 0, 0, 0x80000000]
    codes[0, 0, 4] = 0xAAAAAAAA
    codes[0, 0, 5] = 0x55555555
    qu = rng.integers(0, 16, (B, Hq, D)).astype(np.uint8)
    qu[0, 0] = 15
    qu[0, 1] = 0
    n = np.array([L, L - 7], np.int32)
    d1, p1 = orc.int_dots(codes, qu, n, packed=False)
    d2, p2 = orc.int_dots(codes, qu, n, packed=True)
    assert (d1 == d2).all() and (p1 == p2).all()
    G = Hq // Hkv
    for b in range(B):
        for h in range(Hq):
            ref = _planes_dot_numpy(codes[b, h // G, :n[b]], qu[b, h])
            assert (d1[b, h, :n[b]] == ref).all()
        assert (p1[b, :, :n[b]] == unpack(codes[b, :, :n[b]]).sum(-1)).all()
    assert (d1 <= 15 * np.repeat(p1, G, axis=1)).all()
    assert d1[0, 0, 1] == 15 * 128 and p1[0, 0, 1] == 128 and d1[0, 1, 1] == 0
    assert (d1[1, :, n[1]:] == 0).all()        # beyond n_indexed untouched


def test_o3_int4_quantiser(orc, rot128):
    r32, r64 = rot128
    w = synth.make_workload(1, L=128)
    ck = np.zeros((1, 8, D), np.float32)
    qp = orc.query_prep(w.q, 8, 0, r32, ck)
    q64 = w.q.astype(np.float64)
    np.testing.assert_allclose(qp["qn"], np.linalg.norm(q64, axis=-1), rtol=1e-6)
    qprime = (q64 / np.linalg.norm(q64, axis=-1, keepdims=True)) @ r32.astype(np.float64)
    np.testing.assert_allclose(qp["qprime"], qprime, atol=2e-6)
    np.testing.assert_allclose(np.linalg.norm(qp["qprime"].astype(np.float64), axis=-1), 1.0, atol=1e-5)
    assert qp["qu"].min() == 0 and qp["qu"].max() == 15
    for h in range(32):
        qu, ql, dl = qp["qu"][0, h].astype(np.float64), float(qp["ql"][0, h]), float(qp["delta"][0, h])
        assert ql == qp["qprime"][0, h].min()
        assert dl == pytest.approx((qp["qprime"][0, h].max() - ql) / 15, rel=1e-6)
        assert (qu[np.argmin(qp["qprime"][0, h])] == 0) and (qu[np.argmax(qp["qprime"][0, h])] == 15)
        recon = dl * qu + ql                              # q_bar = Delta*qu + q_l (L524)
        assert np.abs(recon - qp["qprime"][0, h]).max() <= dl / 2 * (1 + 1e-4)
        assert qp["sumq"][0, h] == qu.sum()


def test_o3_degenerate_constant_query(orc):
    I = np.eye(D, dtype=np.float32)
    q = np.full((1, 1, D), 0.5, np.float32)
    qp = orc.query_prep(q, 1, 0, I, np.zeros((1, 1, D), np.float32))
    assert qp["delta"][0, 0] == 0 and (qp["qu"] == 0).all() and qp["sumq"][0, 0] == 0


def test_p7_eq20_equals_direct_and_eq2_identity(orc, rot128):
    r32, r64 = rot128
    w = synth.make_workload(1, L=512, with_cq=True)
    L = 512
    ck = orc.centroid(w.K, w.seq_lens)
    codes, fs, fb = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck, w.c_q)
    sm = 1 / math.sqrt(D)
    scores, qp, dot, pop = orc.estimate_scores(w.q, codes, fs, fb, ck, w.c_q, w.seq_lens, 0, r32, sm)
    G = w.G
    for h in (0, 7, 13, 31):
        g = h // G
        cprime = 2 * unpack(codes[0, g, :L]) - 1                                  # c' = 2c_b - 1
        qbar = float(qp["delta"][0, h]) * qp["qu"][0, h].astype(np.float64) + float(qp["ql"][0, h])
        ip_direct = cprime @ qbar                                                 # Eq.19
        ip20 = (2 * float(qp["delta"][0, h]) * dot[0, h, :L] + 2 * float(qp["ql"][0, h]) * pop[0, g, :L]
                - float(qp["delta"][0, h]) * qp["sumq"][0, h] - D * float(qp["ql"][0, h]))   # Eq.20
        np.testing.assert_allclose(ip20, ip_direct, rtol=0, atol=1e-10)
        S = (float(qp["qn"][0, h]) * fs[0, g, :L].astype(np.float64) * ip_direct + float(qp["q_ck"][0, h])
             + fb[0, h, :L].astype(np.float64) - float(qp["cq_ck"][0, h])) * sm
        np.testing.assert_allclose(scores[0, h, :L], S, rtol=2e-6, atol=1e-6)
        # Eq.2 with the exact cosine reproduces <q,k> for arbitrary centroids
        q64, cq, c_k = w.q[0, h].astype(np.float64), w.c_q[0, h].astype(np.float64), ck[0, g].astype(np.float64)
        k64 = w.K[0, g, :L].astype(np.float64)
        xq, xk = q64 - cq, k64 - c_k
        cos = (xk @ xq) / (np.linalg.norm(xk, axis=1) * np.linalg.norm(xq))
        rhs = np.linalg.norm(xq) * np.linalg.norm(xk, axis=1) * cos + q64 @ c_k + k64 @ cq - cq @ c_k
        np.testing.assert_allclose(rhs, k64 @ q64, rtol=1e-12, atol=1e-10)
        # and the estimate is close to the truth: error std ~ ||xq|| ||xk|| / sqrt(D-1) * sqrt(1/alpha^2-1)
        err = scores[0, h, :L] / sm - k64 @ q64
        bound = np.linalg.norm(xq) * np.linalg.norm(xk, axis=1) * 0.0668 * 1.1
        assert np.abs(err / bound).std() < 1.3 and abs((err / bound).mean()) < 0.25


def test_eq2_bias_terms_from_raw_arrays(orc, rot128):
    """Tight pin of the Eq.2 assembly (Eq.2): with non-zero c_q and a deliberately LARGE c_k (keys
    shifted by +3) the part of the oracle's score that is not the estimated inner product must equal
    <q,c_k> + <c_q,k_t> - <c_q,c_k> computed with numpy in fp64 FROM THE RAW ARRAYS (not from the oracle's query_prep),
    with the KV-head mapping g = h // G spelled out; q_ck / cq_ck of rbq_ref_query_prep against numpy dots."""
    r32, _ = rot128
    w = synth.make_workload(1, L=384, with_cq=True)
    K = (w.K + 3.0).astype(np.float32)                   # large centroid: a wrong sign or KV head moves the score by O(100)
    c_q = (w.c_q + 0.5).astype(np.float32)               # and a query centroid that is not orthogonal to it
    L, G, sm = 384, w.G, 1 / math.sqrt(D)
    ck = orc.centroid(K, w.seq_lens)
    assert np.abs(ck).mean() > 2.5
    codes, fs, fb = orc.encode(K, [0], w.seq_lens, 0, r32, ck, c_q)
    scores, qp, dot, pop = orc.estimate_scores(w.q, codes, fs, fb, ck, c_q, w.seq_lens, 0, r32, sm)
    for h in range(w.Hq):
        g = h // G
        q64, cq64, ck64 = w.q[0, h].astype(np.float64), c_q[0, h].astype(np.float64), ck[0, g].astype(np.float64)
        k64 = K[0, g, :L].astype(np.float64)
        assert float(qp["q_ck"][0, h]) == pytest.approx(q64 @ ck64, rel=1e-6, abs=1e-5)
        assert float(qp["cq_ck"][0, h]) == pytest.approx(cq64 @ ck64, rel=1e-6, abs=1e-5)
        np.testing.assert_allclose(fb[0, h, :L], k64 @ cq64, rtol=2e-6, atol=2e-5)          # f_bias = <c_q, k_t>
        qn = np.linalg.norm(q64 - cq64)
        dl, ql = float(qp["delta"][0, h]), float(qp["ql"][0, h])
        ip20 = 2 * dl * dot[0, h, :L] + 2 * ql * pop[0, g, :L] - dl * int(qp["sumq"][0, h]) - D * ql   # Eq.20 (pinned above)
        est = qn * fs[0, g, :L].astype(np.float64) * ip20
        rest = scores[0, h, :L].astype(np.float64) / sm - est
        want = q64 @ ck64 + k64 @ cq64 - cq64 @ ck64
        scale = np.abs(scores[0, h, :L] / sm).max()
        np.testing.assert_allclose(rest, want, rtol=0, atol=1e-5 * max(scale, np.abs(want).max()))
        # a slip would be visible: each term is far larger than the tolerance
        tol = 1e-5 * max(scale, np.abs(want).max())
        assert min(abs(q64 @ ck64), abs(cq64 @ ck64), np.median(np.abs(k64 @ cq64))) > 300 * tol


def test_estimator_exact_for_codeword_keys_and_grid_queries(orc, rot128):
    """End-to-end pin of O2 -> O3 -> O4 -> O5 against the plain inner product: the estimator
    <c', q_bar> / <c', P^T k_c> (Eq.18) is EXACT when P^T k_c is parallel to its own codeword (|y_j| all equal,
    alpha = 1: L98, L487) and the rotated query lies on the 16-level INT4 grid (Eq.5 L194 then reconstructs it
    exactly).  Then Eq.2 (L86) must give back <q,k> itself for arbitrary c_q, c_k -- every term, sign, the h // G
    mapping and sm_scale are checked against numpy's dot product."""
    r32, r64 = rot128
    rng = np.random.default_rng(42)
    B, Hq, Hkv, L = 1, 8, 2, 64
    G = Hq // Hkv
    P = r32.astype(np.float64)
    ck = (3.0 + rng.standard_normal((B, Hkv, D))).astype(np.float32)
    cq = (0.5 * rng.standard_normal((B, Hq, D))).astype(np.float32)
    s = rng.integers(0, 2, (Hkv, L, D)) * 2.0 - 1.0                       # sign patterns = codewords
    lam = rng.uniform(0.2, 3.0, (Hkv, L, 1))
    x = (lam * s) @ P.T                                                    # x P = lam * s
    K = (ck[0][:, None, :].astype(np.float64) + x).astype(np.float32)[None]
    m = rng.integers(0, 16, (Hq, D)).astype(np.float64)
    m[:, 0], m[:, 1] = 0, 15                                               # both ends of the grid present
    qprime = -0.37 + 0.05 * m
    qprime /= np.linalg.norm(qprime, axis=1, keepdims=True)
    qn = rng.uniform(2.0, 9.0, (Hq, 1))
    q = (cq[0].astype(np.float64) + qn * (qprime @ P.T)).astype(np.float32)[None]
    n = np.array([L], np.int32)
    codes, fs, fb = orc.encode(K, [0], n, 0, r32, ck, cq)
    assert (unpack(codes[0]) == (s > 0)).all()                             # the key's code is its own sign pattern
    sm = 0.25
    scores, qp, _, _ = orc.estimate_scores(q, codes, fs, fb, ck, cq, n, 0, r32, sm)
    assert (qp["qu"][0] == m).all()                                        # the query sits on the INT4 grid
    for h in range(Hq):
        g = h // G
        truth = K[0, g].astype(np.float64) @ q[0, h].astype(np.float64) * sm
        scale = np.linalg.norm(K[0, g].astype(np.float64), axis=1) * np.linalg.norm(q[0, h].astype(np.float64)) * sm
        assert np.abs(scores[0, h, :L] - truth).max() <= 2e-5 * scale.max(), (h, np.abs(scores[0, h, :L] - truth).max())


def _law_samples(orc, c, n_rot, seed):
    """est - c over n_rot Haar rotations for fixed unit k_c, q_c with <k_c,q_c> = c, through the
    oracle's own encode / query_prep / logits chain."""
    rng = np.random.default_rng([7, seed])
    k = np.zeros((1, 1, 1, D), np.float32)
    k[0, 0, 0, 0] = 1.0
    q = np.zeros((1, 1, D), np.float32)
    q[0, 0, 0], q[0, 0, 1] = c, math.sqrt(1 - c * c)
    zero = np.zeros((1, 1, D), np.float32)
    est_f, est_q, alpha = [], [], []
    for _ in range(n_rot):
        r32, _ = orc.rotation_from_gaussian(rng.standard_normal((D, D)))
        codes, fs, _ = orc.encode(k, [0], [1], 0, r32, zero)
        scores, qp, _, _ = orc.estimate_scores(q, codes, fs, None, zero, None, [1], 0, r32, 1.0)
        cp = 2 * unpack(codes[0, 0, :1])[0] - 1
        a_prime = 1.0 / float(fs[0, 0, 0])              # <c', P^T k_c> = ||y||_1 (||x|| = 1)
        est_f.append(float(cp @ qp["qprime"][0, 0].astype(np.float64)) / a_prime * float(qp["qn"][0, 0]))
        est_q.append(float(scores[0, 0, 0]))
        alpha.append(a_prime / math.sqrt(D))
    return np.array(est_f), np.array(est_q), np.array(alpha)


@pytest.mark.parametrize("c", [0.0, 0.3, 0.8])
def test_p3_p4_unbiasedness_law(orc, c):
    n = 4096
    est_f, est_q, alpha = _law_samples(orc, c, n, int(c * 10))
    # P4: closed form E[alpha] (golden: tests/golden/alpha_closed_form.txt, from the density at L558)
    gold = dict(l.split()[:2] for l in (GOLD / "alpha_closed_form.txt").read_text().splitlines()
                if l and not l.startswith("#"))
    e_alpha = math.sqrt(D) * math.exp(gammaln(D / 2) - gammaln((D + 1) / 2)) / math.sqrt(math.pi)
    assert e_alpha == pytest.approx(float(gold["128"]), abs=1e-6)
    assert abs(alpha.mean() - e_alpha) < 4 * alpha.std() / math.sqrt(n)
    assert 0.015 < alpha.std() < 0.022
    # P3 float query: z = (est-c) alpha / (sqrt(1-alpha^2) sqrt(1-c^2)) ~ p_{D-1}: mean 0, var 1/(D-1)
    z = (est_f - c) * alpha / (np.sqrt(1 - alpha ** 2) * math.sqrt(1 - c * c))
    assert abs((est_f - c).mean()) < 4 * (est_f - c).std() / math.sqrt(n)
    assert 0.9 < z.var() * (D - 1) < 1.1
    assert (np.abs(z) <= 2.6 / math.sqrt(D - 1)).mean() >= 0.985
    assert np.abs(z).max() <= 1.0
    # INT4 query (Thm A.2): still centred (deterministic rounding adds < Delta-sized bias), var +<=20 %
    se = (est_q - c).std() / math.sqrt(n)
    assert abs((est_q - c).mean()) < 4 * se + 2e-3
    assert 0.9 < (est_q - c).var() / (est_f - c).var() < 1.2
    # |err| = O(1/sqrt(D)) w.h.p. (Eq.14)
    assert (np.abs(est_q - c) < 3.5 / math.sqrt(D)).mean() > 0.999


def test_space_overhead_formula():
    # (D/8 + B_alpha)/(2*D*2) = 3.5 % at D=128, FP16 KV, FP16 alpha
    line = [l for l in (GOLD / "alpha_closed_form.txt").read_text().splitlines() if l.startswith("space")][0]
    assert (D / 8 + 2) / (2 * D * 2) == pytest.approx(float(line.split()[1]), abs=5e-4)
