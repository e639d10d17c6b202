"""Pins for oracle O1 (rotation) and O2 (Alg.1 index construction).  CPU only.

P1 orthogonality (BASELINE.json: P^T P = I to 1e-5), agreement with numpy's QR up to column
signs, WH variant exactly orthogonal; P8 encode invariants (Eq.18):
0 < alpha <= 1, alpha = 1/sqrt(D) for a key along one rotated axis, scale invariance of the
code, f_scale = ||x||^2/||y||_1; codes against an independent numpy fp64 rotation; bit order
(L270: 32 consecutive dims per 32-bit word, little-endian, R10).
"""
import math

import numpy as np
import pytest

from paper_2606_31519_b200 import synth

D = 128


def unpack(codes):
    """uint32 [..., D/32] -> {0,1} [..., D] (dim j = word j//32, bit j%32)."""
    sh = np.arange(32, dtype=np.uint32)
    bits = (codes[..., :, None] >> sh) & 1
    return bits.reshape(codes.shape[:-1] + (codes.shape[-1] * 32,)).astype(np.int64)


def test_p1_orthogonality_fp32(rot128):
    r32, r64 = rot128
    assert np.abs(r32.astype(np.float64).T @ r32.astype(np.float64) - np.eye(D)).max() <= 1e-5
    assert np.abs(r64.T @ r64 - np.eye(D)).max() <= 1e-13
    assert np.abs(r64 @ r64.T - np.eye(D)).max() <= 1e-13


def test_p1_matches_numpy_qr_up_to_signs(rot128):
    _, r64 = rot128
    A = synth.rotation_gaussian(D)
    Q, R = np.linalg.qr(A)
    Q = Q * np.sign(np.diag(R))          # the factor with positive diagonal: unique => Haar
    assert np.abs(Q - r64).max() <= 1e-11
    # and it really is a QR factor of A with an upper-triangular, positive-diagonal R
    Rt = r64.T @ A
    assert np.abs(np.tril(Rt, -1)).max() <= 1e-11
    assert (np.diag(Rt) > 0).all()


def test_p1_haar_sign_convention_changes_with_input(orc):
    # flipping the sign of column j of A flips column j of Q only (positive-diagonal convention)
    A = synth.rotation_gaussian(D)
    _, q0 = orc.rotation_from_gaussian(A)
    A2 = A.copy()
    A2[:, 5] *= -1
    _, q1 = orc.rotation_from_gaussian(A2)
    diff = np.abs(q0 - q1).max(axis=0)
    assert diff[5] > 1e-3 and np.abs(q0[:, 5] + q1[:, 5]).max() < 1e-11
    assert np.delete(diff, 5).max() < 1e-11


def test_wh_rotation_orthogonal_and_matches_fwht(orc):
    s = synth.wh_sign_vector(D)
    R = orc.rotation_wh(s).astype(np.float64)
    assert np.abs(R.T @ R - np.eye(D)).max() <= 2e-7       # only the 1/sqrt(D) rounding
    x = np.random.default_rng(3).standard_normal(D).astype(np.float32)
    u = orc.fwht(s * x)                                     # unscaled butterflies
    # Sylvester Hadamard written out independently
    H = np.array([[(-1) ** bin(i & j).count("1") for j in range(D)] for i in range(D)], np.float64)
    np.testing.assert_allclose(u, H @ (s * x).astype(np.float64), rtol=0, atol=1e-4)
    np.testing.assert_allclose(u / math.sqrt(D), x.astype(np.float64) @ R, atol=1e-5)
    # involution: H(Hx) = D x
    np.testing.assert_allclose(orc.fwht(orc.fwht(x)), D * x, rtol=1e-6, atol=1e-4)


def _encode_one(orc, x, rot, kind=0):
    K = np.zeros((1, 1, 1, D), np.float32)
    K[0, 0, 0] = x
    codes, fs, _ = orc.encode(K, [0], [1], kind, rot, np.zeros((1, 1, D), np.float32))
    return codes[0, 0, 0], float(fs[0, 0, 0])


def test_p8_axis_key_has_min_alpha(orc, rot128):
    r32, _ = rot128
    lam = 2.5
    j = 17
    # y = x R; x = lam * (row... ) we need y = lam * e_j => x = lam * R[:, j]^T^-1 = lam * R[j, :]^T? y_j' = sum_i x_i R[i][j']
    # with x = lam * R[:, j] (column j of R): y = lam * R^T R[:, j] = lam * e_j (orthogonality)
    x = (lam * r32[:, j]).astype(np.float32)
    code, fs = _encode_one(orc, x, r32)
    bits = unpack(code[None])[0]
    assert bits[j] == 1
    # alpha' = ||y||_1/||x||_2 ; alpha = alpha'/sqrt(D) ; for y ~ lam*e_j (+1e-7 leakage) alpha ~ 1/sqrt(D)
    n2 = float(np.dot(x.astype(np.float64), x.astype(np.float64)))
    alpha = (n2 / fs) / math.sqrt(n2) / math.sqrt(D)
    assert abs(alpha - 1 / math.sqrt(D)) < 2e-5


def test_p8_alpha_range_and_scale_invariance(orc, rot128):
    r32, r64 = rot128
    rng = np.random.default_rng(11)
    for _ in range(50):
        x = rng.standard_normal(D).astype(np.float32) * rng.uniform(0.1, 30)
        code, fs = _encode_one(orc, x, r32)
        n = np.linalg.norm(x.astype(np.float64))
        alpha = (n * n / fs) / n / math.sqrt(D)
        assert 0 < alpha <= 1 + 1e-6
        code2, fs2 = _encode_one(orc, (4.0 * x).astype(np.float32), r32)   # power of two: exact scaling
        assert (code == code2).all()
        assert fs2 == pytest.approx(4.0 * fs, rel=1e-7)
        # closed form in fp64 with an independent rotation product
        y = x.astype(np.float64) @ r32.astype(np.float64)
        assert fs == pytest.approx(n * n / np.abs(y).sum(), rel=2e-6)


def test_p8_alpha_one_iff_equal_magnitudes(orc):
    # identity "rotation": y = x; |y_j| all equal => alpha = 1 exactly
    I = np.eye(D, dtype=np.float32)
    x = np.where(np.random.default_rng(5).integers(0, 2, D) > 0, 0.75, -0.75).astype(np.float32)
    code, fs = _encode_one(orc, x, I)
    n2 = D * 0.75 ** 2
    assert fs == pytest.approx(n2 / (D * 0.75), rel=1e-7)           # ||x||^2/||y||_1
    alpha = (n2 / fs) / math.sqrt(n2) / math.sqrt(D)
    assert alpha == pytest.approx(1.0, abs=1e-6)
    assert (unpack(code[None])[0] == (x > 0)).all()


def test_bit_order_and_sign_of_zero(orc):
    I = np.eye(D, dtype=np.float32)
    x = np.zeros(D, np.float32)
    x[0], x[31], x[32], x[127], x[64] = 1, 2, 3, 4, -5     # zeros elsewhere -> bit 0 (L485)
    code, _ = _encode_one(orc, x, I)
    assert code[0] == (1 | (1 << 31)) and code[1] == 1 and code[2] == 0 and code[3] == (1 << 31)
    # zero vector: f_scale = 0 (R15), all bits 0
    code0, fs0 = _encode_one(orc, np.zeros(D, np.float32), I)
    assert (code0 == 0).all() and fs0 == 0.0


def test_codes_match_independent_fp64_rotation_cfg0(orc, rot128):
    r32, _ = rot128
    w = synth.make_workload(0, L=1024 + 37)
    ck = orc.centroid(w.K, w.seq_lens)
    L = int(w.seq_lens[0])
    np.testing.assert_allclose(ck[0, 0], w.K[0, 0, :L].astype(np.float64).mean(axis=0), rtol=1e-6, atol=1e-7)
    codes, fs, _ = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck)
    x = w.K[0, 0, :L].astype(np.float64) - ck[0, 0].astype(np.float64)
    y = x @ r32.astype(np.float64)
    bits = unpack(codes[0, 0, :L])
    safe = np.abs(y) > 1e-5 * np.linalg.norm(x, axis=1, keepdims=True)
    assert ((bits == (y > 0)) | ~safe).all()
    assert safe.mean() > 0.999
    np.testing.assert_allclose(fs[0, 0, :L], (x * x).sum(1) / np.abs(y).sum(1), rtol=3e-6)
    # mean alpha over real keys ~ 0.80 (closed form E[alpha])
    alpha = np.abs(y).sum(1) / np.linalg.norm(x, axis=1) / math.sqrt(D)
    assert 0.78 < alpha[4:].mean() < 0.82
    # tokens beyond seq_len untouched
    assert (codes[0, 0, L:] == 0).all() and (fs[0, 0, L:] == 0).all()


def test_wh_encode_matches_dense_encode_of_materialised_matrix(orc):
    s = synth.wh_sign_vector(D)
    R = orc.rotation_wh(s)
    w = synth.make_workload(0, L=512)
    ck = orc.centroid(w.K, w.seq_lens)
    c_wh, f_wh, _ = orc.encode(w.K, [0], w.seq_lens, 1, s, ck)
    c_de, f_de, _ = orc.encode(w.K, [0], w.seq_lens, 0, R, ck)
    L = 512
    x = w.K[0, 0, :L].astype(np.float64) - ck[0, 0]
    y = x @ R.astype(np.float64)
    safe = np.abs(y) > 1e-5 * np.linalg.norm(x, axis=1, keepdims=True)
    assert ((unpack(c_wh[0, 0, :L]) == unpack(c_de[0, 0, :L])) | ~safe).all()
    np.testing.assert_allclose(f_wh[0, 0, :L], f_de[0, 0, :L], rtol=3e-6)


def test_f_bias_is_cq_dot_k(orc, rot128):
    r32, _ = rot128
    w = synth.make_workload(1, L=256, with_cq=True)
    ck = orc.centroid(w.K, w.seq_lens)
    _, _, fb = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck, w.c_q)
    G = w.G
    for h in (0, 5, 31):
        ref = w.K[0, h // G, :256].astype(np.float64) @ w.c_q[0, h].astype(np.float64)
        np.testing.assert_allclose(fb[0, h, :256], ref, rtol=1e-5, atol=1e-4)


def test_factors_f16_rounding_and_logit_bound(orc, rot128):
    """O2c (PAPER.md:L752 FP16 factors; L756-766 space accounting): the rounded factor equals numpy's float32 -> float16 ->
    float32 conversion (an independent RNE implementation) bit for bit, is idempotent, moves each factor by at most 2^-11
    relative, and therefore moves the ESTIMATED part of every logit by at most 2^-11 relative (the Eq.2 bias terms do
    not involve the factor); the space overhead with 2-byte factors is the paper's 3.5 %."""
    import math
    from paper_2606_31519_b200 import synth
    r32, _ = rot128
    w = synth.make_workload(1, L=777)
    ck = orc.centroid(w.K, w.seq_lens)
    codes, fs, _ = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck)
    fs16 = orc.round_factors_f16(fs)
    assert (fs16.view(np.uint32) == fs.astype(np.float16).astype(np.float32).view(np.uint32)).all()
    assert (orc.round_factors_f16(fs16).view(np.uint32) == fs16.view(np.uint32)).all()
    n = int(w.seq_lens[0])
    live = fs[0, :, :n]
    assert (np.abs(fs16[0, :, :n] - live) <= 2.0 ** -11 * np.abs(live)).all() and (fs16 != fs).any()
    sm = 1 / math.sqrt(128)
    s32, qp, dot, pop = orc.estimate_scores(w.q, codes, fs, None, ck, None, w.seq_lens, 0, r32, sm)
    s16, _, _, _ = orc.estimate_scores(w.q, codes, fs16, None, ck, None, w.seq_lens, 0, r32, sm)
    const = (qp["q_ck"] - qp["cq_ck"])[..., None].astype(np.float64) * sm        # Eq.2 terms that carry no factor
    est = s32[..., :n].astype(np.float64) - const
    assert (np.abs(s16[..., :n].astype(np.float64) - s32[..., :n]) <= 2.0 ** -11 * np.abs(est) * (1 + 1e-3) + 1e-6).all()
    assert (128 / 8 + 2) / (2 * 128 * 2) == pytest.approx(0.035, abs=5e-4)
