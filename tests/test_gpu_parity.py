"""GPU-vs-oracle parity of every stage of the RaBitQCache decode path, through the C ABI
(include/rbq.h -> paper_2606_31519_b200.binding).  Stage-isolated: each GPU stage is fed the
ORACLE's upstream arrays so one stage's legal rounding cannot cascade; the chained tests are in
test_gpu_chained.py.

Tolerances (BASELINE.json north_star): codes / factors / INT4 query codes / integer dots
bit-exact; logits 1e-5 relative; Top-p sets identical up to boundary tokens (1e-6); attention
1e-2 rel + 2e-2 abs for bf16 inputs (1e-4 / 1e-4 for fp32).
"""
import numpy as np
import pytest

from tests import gpu_util as U

pytestmark = pytest.mark.gpu

ROT_DENSE, ROT_WH = 0, 1

# (name, cfg, kwargs): sizes the oracle finishes in seconds; ragged tails on purpose
CASES = {
    "cfg0": (0, dict()),                                      # B=1, Hq=Hkv=1, L=4096, fp32 (BASELINE config 0 in full)
    "cfg0_cq": (0, dict(with_cq=True)),                       # same with a non-zero query centroid (Eq.2 for any c_q)
    "cfg1_small": (1, dict(L=5003)),                          # GQA 4:1, bf16, ragged L
    "cfg2_small": (2, dict(L=6150, n_heavy=32)),              # temperature knob
    "cfg3_small": (3, dict(L=3001, B=3)),                     # batch of ragged lengths in [L/4, L]
}


def get_case(name):
    cfg, kw = CASES[name]
    return U.workload(cfg, **kw)


@pytest.fixture(scope="module")
def wh_signs():
    from paper_2606_31519_b200 import synth
    return synth.wh_sign_vector(128)


def _rot(kind, rot128, wh_signs):
    return rot128[0] if kind == ROT_DENSE else wh_signs


# ---- S1: Alg.1 index construction -----------------------------------------------------------------------
@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("name", ["cfg0", "cfg0_cq", "cfg1_small", "cfg3_small"])
def test_encode_keys_bit_exact(orc, rot128, wh_signs, name, kind):
    import torch
    w = get_case(name)
    with_cq = w.c_q is not None
    rot = _rot(kind, rot128, wh_signs)
    o = U.oracle_index(orc, w, rot, kind, with_cq)
    c = U.make_cache(w, rot, rot_kind=kind, with_cq=with_cq)
    c.codes.fill_(-1)
    c.encode_keys(U.to_dev(w.seq_lens))
    torch.cuda.synchronize()
    assert (c.n_indexed.cpu().numpy() == w.seq_lens).all() and (c.n_total.cpu().numpy() == w.seq_lens).all()
    ck = c.c_k.cpu().numpy()
    assert (ck.view(np.uint32) == o["c_k"].view(np.uint32)).all(), "centroid differs"
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    for b in range(w.B):
        n = int(w.seq_lens[b])
        assert (codes[b, :, :n] == o["codes"][b, :, :n]).all(), f"codes differ (seq {b})"
        assert (fs[b, :, :n].view(np.uint32) == o["f_scale"][b, :, :n].view(np.uint32)).all(), "f_scale differs"
        assert (codes[b, :, n:] == 0xFFFFFFFF).all(), "encode wrote beyond seq_len"
        if with_cq:
            fb = c.f_bias.cpu().numpy()
            assert (fb[b, :, :n].view(np.uint32) == o["f_bias"][b, :, :n].view(np.uint32)).all(), "f_bias differs"
    c.close()


def test_encode_ck_given_and_zero_key(orc, rot128):
    """RBQ_CK_GIVEN keeps the caller's centroid; a key equal to c_k gives code 0 and f_scale 0 (R: C18)."""
    import torch
    from paper_2606_31519_b200 import binding as rb
    w = U.workload(0, L=300)
    ck = (0.25 * np.random.default_rng(5).standard_normal((1, 1, 128))).astype(np.float32)
    K = w.K.copy()
    K[0, 0, 17] = ck[0, 0]
    codes, fs, _ = orc.encode(K, np.zeros(1, np.int32), w.seq_lens, ROT_DENSE, rot128[0], ck)
    c = U.make_cache(w, rot128[0])
    c.K.copy_(U.to_dev(K))
    c.c_k.copy_(U.to_dev(ck))
    c.encode_keys(U.to_dev(w.seq_lens), flags=rb.RBQ_CK_GIVEN)
    torch.cuda.synchronize()
    n = int(w.seq_lens[0])
    assert (c.c_k.cpu().numpy() == ck).all()
    assert (c.codes.cpu().numpy().view(np.uint32)[0, 0, :n] == codes[0, 0, :n]).all()
    got = c.f_scale.cpu().numpy()[0, 0, :n]
    assert (got.view(np.uint32) == fs[0, 0, :n].view(np.uint32)).all()
    assert got[17] == 0.0 and (c.codes.cpu().numpy()[0, 0, 17] == 0).all()
    c.close()


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("name", ["cfg1_small", "cfg3_small"])
def test_encode_fast_guard_band(orc, rot128, wh_signs, name, kind):
    """RBQ_ENC_FAST (tensor-core rotation, bf16 hi/lo split): a code bit may differ from the oracle's only where the
    fp64 rotated coordinate satisfies |y_j| <= 1e-5 ||x|| (expected fraction ~9e-5, fail above 3e-4); f_scale within
    1e-5 relative."""
    _check_encode_fast(orc, _rot(kind, rot128, wh_signs), get_case(name), kind)


def test_encode_fast_many_tiles(orc, rot128):
    """The tcgen05 encode kernel over several 128-token tiles per CTA and pipeline group (double-buffered accumulators,
    mbarrier phases, register prefetch), a ragged last tile, and a KV head whose keys are all identical (x = 0 for every
    token: zero codes and zero factors, Alg.1 with ||x|| = 0)."""
    w = U.workload(1, L=40077)
    w.K[0, 0, :, :] = w.K[0, 0, :1, :]
    _check_encode_fast(orc, rot128[0], w)


def _check_encode_fast(orc, rot, w, kind=ROT_DENSE):
    import torch
    from paper_2606_31519_b200 import binding as rb
    o = U.oracle_index(orc, w, rot, kind)
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)), rot_kind=kind,
                       enc_mode=rb.RBQ_ENC_FAST)
    c.K.copy_(U.to_dev(w.K, torch.bfloat16))
    c.encode_keys(U.to_dev(w.seq_lens))
    torch.cuda.synchronize()
    assert np.array_equal(c.c_k.cpu().numpy().view(np.uint32), o["c_k"].view(np.uint32))
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    P = (rot if kind == ROT_DENSE else orc.rotation_wh(rot)).astype(np.float64)
    n_bits = n_diff = 0
    for b in range(w.B):
        n = int(w.seq_lens[b])
        for g in range(w.Hkv):
            x = w.K[b, g, :n].astype(np.float64) - o["c_k"][b, g].astype(np.float64)
            y = x @ P
            xn = np.linalg.norm(x, axis=1, keepdims=True)
            diff = codes[b, g, :n] ^ o["codes"][b, g, :n]                       # [n, 4] words
            bits = ((diff[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(n, 128).astype(bool)
            assert (np.abs(y)[bits] <= 1e-5 * np.broadcast_to(xn, y.shape)[bits]).all(), "code bit differs outside the guard band"
            n_bits += bits.size
            n_diff += int(bits.sum())
            ref = o["f_scale"][b, g, :n].astype(np.float64)
            assert (np.abs(fs[b, g, :n] - ref) <= 1e-5 * np.abs(ref)).all(), "f_scale outside 1e-5 relative"
            zero = (xn[:, 0] == 0.0)
            assert (codes[b, g, :n][zero] == 0).all() and (fs[b, g, :n][zero] == 0.0).all()
    assert n_diff <= 3e-4 * n_bits, f"{n_diff} of {n_bits} bits differ"
    c.close()


# ---- S3: query prep + INT4 quantisation -------------------------------------------------------------------
@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("name", ["cfg0", "cfg0_cq", "cfg1_small", "cfg3_small"])
def test_query_quantize_bit_exact(orc, rot128, wh_signs, name, kind):
    import torch
    w = get_case(name)
    with_cq = w.c_q is not None
    rot = _rot(kind, rot128, wh_signs)
    c_k = orc.centroid(w.K, w.seq_lens)
    qp = orc.query_prep(w.q, w.Hkv, kind, rot, c_k, w.c_q)
    c = U.make_cache(w, rot, rot_kind=kind, with_cq=with_cq, upload_kv=False)
    c.c_k.copy_(U.to_dev(c_k))
    qu = torch.zeros(w.B, w.Hq, 128, dtype=torch.uint8, device="cuda")
    par = torch.zeros(w.B, w.Hq, 6, dtype=torch.float32, device="cuda")
    c.query_quantize(U.to_dev(w.q, U.torch_dtype(w)), qu, par)
    torch.cuda.synchronize()
    assert (qu.cpu().numpy() == qp["qu"]).all(), "INT4 query codes differ"
    par = par.cpu().numpy()
    for i, key in enumerate(["qn", "ql", "delta"]):
        assert (par[..., i].view(np.uint32) == qp[key].view(np.uint32)).all(), key
    assert (par[..., 3] == qp["sumq"]).all()
    assert (par[..., 4].view(np.uint32) == qp["q_ck"].view(np.uint32)).all()
    assert (par[..., 5].view(np.uint32) == qp["cq_ck"].view(np.uint32)).all()
    c.close()


def test_query_degenerate_constant_rotated_query(orc):
    """q_r == q_l (R5): with P = I and q = const vector, Delta = 0 and every INT4 code is 0."""
    import torch
    w = U.workload(0, L=64)
    eye = np.eye(128, dtype=np.float32)
    q = np.full((1, 1, 128), 0.5, np.float32)
    c_k = np.zeros((1, 1, 128), np.float32)
    qp = orc.query_prep(q, 1, ROT_DENSE, eye, c_k)
    assert qp["delta"][0, 0] == 0.0 and (qp["qu"] == 0).all()
    c = U.make_cache(w, eye, upload_kv=False)
    qu = torch.full((1, 1, 128), 9, dtype=torch.uint8, device="cuda")
    par = torch.zeros(1, 1, 6, device="cuda")
    c.query_quantize(U.to_dev(q), qu, par)
    torch.cuda.synchronize()
    assert (qu.cpu().numpy() == 0).all()
    par = par.cpu().numpy()
    assert par[0, 0, 2] == 0.0 and par[0, 0, 1] == qp["ql"][0, 0] and par[0, 0, 0] == qp["qn"][0, 0]
    c.close()


# ---- S4: Int4_Dot_Binary -----------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg0", "cfg1_small", "cfg2_small", "cfg3_small"])
def test_int4_dot_binary_bit_exact(orc, rot128, name):
    import torch
    w = get_case(name)
    o = U.oracle_full(orc, w, rot128[0])
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    dot = torch.full((w.B, w.Hq, w.Lcap), -7, dtype=torch.int32, device="cuda")
    pop = torch.full((w.B, w.Hkv, w.Lcap), -7, dtype=torch.int32, device="cuda")
    c.int4_dot_binary(U.to_dev(w.q, U.torch_dtype(w)), dot, pop)
    torch.cuda.synchronize()
    dot, pop = dot.cpu().numpy(), pop.cpu().numpy()
    for b in range(w.B):
        n = int(w.seq_lens[b])
        assert (dot[b, :, :n] == o["dot"][b, :, :n]).all(), "integer dot differs"
        assert (pop[b, :, :n] == o["pop"][b, :, :n]).all(), "popcount differs"
        assert (dot[b, :, n:] == -7).all() and (pop[b, :, n:] == -7).all(), "wrote beyond n_indexed"
    c.close()


def test_int4_dot_binary_adversarial_codes(orc, rot128):
    """all-0, all-1, single-bit, alternating and random codes against random INT4 queries (P2)."""
    import torch
    rng = np.random.default_rng(11)
    w = U.workload(1, L=1500)
    o = U.oracle_index(orc, w, rot128[0])
    L = int(w.seq_lens[0])
    codes = rng.integers(0, 2 ** 32, (w.B, w.Hkv, w.Lcap, 4), dtype=np.uint64).astype(np.uint32)
    codes[:, :, 0] = 0
    codes[:, :, 1] = 0xFFFFFFFF
    codes[:, :, 2] = 0xAAAAAAAA
    codes[:, :, 3] = 0x55555555
    for j in range(128):
        codes[:, :, 4 + j] = 0
        codes[:, :, 4 + j, j // 32] = np.uint32(1) << np.uint32(j % 32)
    o["codes"] = codes
    qp = orc.query_prep(w.q, w.Hkv, ROT_DENSE, rot128[0], o["c_k"])
    d_ref, p_ref = orc.int_dots(codes, qp["qu"], w.seq_lens)
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    dot = torch.zeros(w.B, w.Hq, w.Lcap, dtype=torch.int32, device="cuda")
    pop = torch.zeros(w.B, w.Hkv, w.Lcap, dtype=torch.int32, device="cuda")
    c.int4_dot_binary(U.to_dev(w.q, U.torch_dtype(w)), dot, pop)
    torch.cuda.synchronize()
    assert (dot.cpu().numpy()[..., :L] == d_ref[..., :L]).all()
    assert (pop.cpu().numpy()[..., :L] == p_ref[..., :L]).all()
    # single-bit codes read back the INT4 query itself
    assert (dot.cpu().numpy()[0, :, 4:132] == qp["qu"][0]).all()
    c.close()


# ---- S5: logits ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("name", ["cfg0", "cfg0_cq", "cfg1_small", "cfg2_small", "cfg3_small"])
def test_estimate_scores(orc, rot128, wh_signs, name, kind):
    import torch
    w = get_case(name)
    with_cq = w.c_q is not None
    rot = _rot(kind, rot128, wh_signs)
    o = U.oracle_full(orc, w, rot, kind, with_cq)
    c = U.make_cache(w, rot, rot_kind=kind, with_cq=with_cq, upload_kv=False)
    U.load_index(c, o)
    scores = torch.full((w.B, w.Hq, w.Lcap), 12345.0, device="cuda")
    c.estimate_scores(U.to_dev(w.q, U.torch_dtype(w)), scores)
    torch.cuda.synchronize()
    s = scores.cpu().numpy()
    U.assert_logits_close(s, o["scores"], w.seq_lens, w.Hq)
    for b in range(w.B):
        assert (s[b, :, int(w.seq_lens[b]):] == 12345.0).all(), "wrote beyond n_indexed"
    c.close()


# ---- S6: Top-p ---------------------------------------------------------------------------------------------
def _run_topp(c, scores_np, p):
    import torch
    sel_idx, sel_cnt = c.new_sel()
    sel_idx.fill_(-1)
    c.topp_select(U.to_dev(scores_np), p, sel_idx, sel_cnt)
    torch.cuda.synchronize()
    return sel_idx.cpu().numpy(), sel_cnt.cpu().numpy()


@pytest.mark.parametrize("p", [0.8, 0.9, 0.95])
@pytest.mark.parametrize("name", ["cfg0", "cfg1_small", "cfg2_small", "cfg3_small"])
def test_topp_select_oracle_scores(orc, rot128, name, p):
    w = get_case(name)
    o = U.oracle_full(orc, w, rot128[0], p=p)
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    idx, cnt = _run_topp(c, o["scores"], p)
    n_boundary = 0
    for b in range(w.B):
        n = int(w.seq_lens[b])
        for h in range(w.Hq):
            g = idx[b, h, :cnt[b, h]]
            assert (np.diff(g) > 0).all(), "sel_idx not ascending"
            assert g.size == 0 or (g.min() >= 0 and g.max() < n)
            n_boundary += U.assert_topp_row(o["scores"][b, h, :n], g, o["sel_idx"][b, h, :o["sel_cnt"][b, h]], p)
            assert (idx[b, h, cnt[b, h]:n] == -1).all() or cnt[b, h] == n
    assert n_boundary <= 2 * w.B * w.Hq
    c.close()


def test_topp_edge_rows(orc, rot128):
    """ties (lowest index wins), all-equal rows, one-token and empty sequences, p >= 1, tiny p, huge spread."""
    rng = np.random.default_rng(21)
    w = U.workload(3, L=2000, B=4)                     # 4 sequences x 32 heads
    rows, L = w.B * w.Hq, w.Lcap
    assert L >= 1400
    n_seq = np.array([L, 1, 0, min(777, L)], np.int32)
    scores = (rng.standard_normal((w.B, w.Hq, L)) * rng.uniform(0.3, 8.0, (w.B, w.Hq, 1))).astype(np.float32)
    scores[0, 3, :50] = scores[0, 3, 0]                # a block of exact ties
    scores[0, 4] = 1.25                                # all equal
    scores[0, 5, 100:1200] = 7.0                       # many ties at the top
    scores[0, 6] = np.round(scores[0, 6])              # heavy duplication everywhere
    scores[0, 7, 10] = 300.0                           # one dominant token (others underflow)
    scores[0, 8] *= 40.0                               # huge dynamic range
    scores[3, 2, :] = -1e30                         # all equal, very negative
    o = dict(codes=np.zeros((w.B, w.Hkv, L, 4), np.uint32), f_scale=np.zeros((w.B, w.Hkv, L), np.float32),
             c_k=np.zeros((w.B, w.Hkv, 128), np.float32), n_indexed=n_seq, n_total=n_seq)
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    n_rows = np.repeat(n_seq, w.Hq)
    for p in (0.02, 0.5, 0.9, 0.999, 1.0):
        ref_idx, ref_cnt = orc.topp(scores.reshape(rows, L), n_rows, p)
        ref_idx, ref_cnt = ref_idx.reshape(w.B, w.Hq, L), ref_cnt.reshape(w.B, w.Hq)
        idx, cnt = _run_topp(c, scores, p)
        for b in range(w.B):
            n = int(n_seq[b])
            for h in range(w.Hq):
                if n == 0:
                    assert cnt[b, h] == 0
                    continue
                g = idx[b, h, :cnt[b, h]]
                assert (np.diff(g) > 0).all() and g.min() >= 0 and g.max() < n
                U.assert_topp_row(scores[b, h, :n], g, ref_idx[b, h, :ref_cnt[b, h]], p)
        if p < 1.0:
            # exact ties: the lowest indices are the ones kept (R8)
            k = ref_cnt[0, 4]
            assert cnt[0, 4] == k and (idx[0, 4, :k] == np.arange(k)).all()
        else:
            assert (cnt[0] == L).all() and (idx[0, 0, :L] == np.arange(L)).all()
    c.close()


@pytest.mark.parametrize("B,L", [(1, 40000), (2, 3000), (8, 3000), (16, 2100), (3, 90)])
def test_topp_cluster_sizes(orc, rot128, B, L):
    """Cluster sizes 4 / 2 / 1 / 1 / 1 of the Top-p kernel (chosen from the row count and the row length; 8 CTAs per row
    is what the single-row config-0 cases run; 2 CTAs per row with more rows than SMs is the config-3 case of
    test_gpu_fullsize.py), rows shorter than one bitmap word per CTA, and the fused step without index lists
    (sel_idx = NULL)."""
    import torch
    rng = np.random.default_rng(5 + B)
    w = U.workload(3, L=L, B=B)
    rows, Lc = w.B * w.Hq, w.Lcap
    n_seq = w.seq_lens.copy()
    scores = (rng.standard_normal((w.B, w.Hq, Lc)) * rng.uniform(0.5, 6.0, (w.B, w.Hq, 1))).astype(np.float32)
    scores[:, 0, :] = np.round(scores[:, 0, :] * 2) / 2            # heavy ties
    o = dict(codes=np.zeros((w.B, w.Hkv, Lc, 4), np.uint32), f_scale=np.zeros((w.B, w.Hkv, Lc), np.float32),
             c_k=np.zeros((w.B, w.Hkv, 128), np.float32), n_indexed=n_seq, n_total=n_seq)
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    for p in (0.5, 0.9):
        ref_idx, ref_cnt = orc.topp(scores.reshape(rows, Lc), np.repeat(n_seq, w.Hq), p)
        ref_idx, ref_cnt = ref_idx.reshape(w.B, w.Hq, Lc), ref_cnt.reshape(w.B, w.Hq)
        idx, cnt = _run_topp(c, scores, p)
        for b in range(w.B):
            n = int(n_seq[b])
            for h in range(w.Hq):
                g = idx[b, h, :cnt[b, h]]
                assert (np.diff(g) > 0).all() and g.min() >= 0 and g.max() < n
                U.assert_topp_row(scores[b, h, :n], g, ref_idx[b, h, :ref_cnt[b, h]], p)
    c.close()


@pytest.mark.parametrize("B,L", [(1, 5000), (2, 40000), (1, 131072)])
def test_topp_alg3_selector(orc, rot128, B, L):
    """rbq_topp_select_alg3 (the paper's Alg.3) against the oracle's Alg.3 on fp64 softmax probabilities:
    identical masks (a mismatch is tolerated only for tokens within 1e-9 relative of the boundary probability), the
    mask is a threshold set whose mass reaches p and is minimal up to ties, iteration counts agree, p >= 1 selects all."""
    import torch
    rng = np.random.default_rng(11 + L)
    w = U.workload(3, L=L, B=B)
    rows, Lc = w.B * w.Hq, w.Lcap
    n_seq = w.seq_lens.copy()
    scores = (rng.standard_normal((w.B, w.Hq, Lc)) * rng.uniform(0.5, 6.0, (w.B, w.Hq, 1))).astype(np.float32)
    scores[:, 0, :] = np.round(scores[:, 0, :] * 2) / 2            # heavy ties: Alg.3 keeps every tied token
    o = dict(codes=np.zeros((w.B, w.Hkv, Lc, 4), np.uint32), f_scale=np.zeros((w.B, w.Hkv, Lc), np.float32),
             c_k=np.zeros((w.B, w.Hkv, 128), np.float32), n_indexed=n_seq, n_total=n_seq)
    c = U.make_cache(w, rot128[0], upload_kv=False)
    U.load_index(c, o)
    sc_dev = U.to_dev(scores)
    heads = range(w.Hq) if L <= 40000 else (0, 1, w.Hq - 1)
    for p in (np.float32(0.5), np.float32(0.9)):
        sel_idx, sel_cnt = c.new_sel()
        sel_idx.fill_(-1)
        iters = torch.zeros((w.B, w.Hq), dtype=torch.int32, device="cuda")
        c.topp_select_alg3(sc_dev, float(p), sel_idx, sel_cnt, iters)
        torch.cuda.synchronize()
        idx, cnt, its = sel_idx.cpu().numpy(), sel_cnt.cpu().numpy(), iters.cpu().numpy()
        for b in range(w.B):
            n = int(n_seq[b])
            for h in heads:
                s64 = scores[b, h, :n].astype(np.float64)
                e = np.exp(s64 - s64.max())
                prob = e / e.sum()
                ref_mask, ref_it = orc.topp_alg3(prob, float(p))
                g = idx[b, h, :cnt[b, h]]
                assert (np.diff(g) > 0).all() and g.min() >= 0 and g.max() < n
                mask = np.zeros(n, bool)
                mask[g] = True
                if not (mask == ref_mask).all():
                    edge = prob[ref_mask].min()
                    diff = mask != ref_mask
                    assert (np.abs(prob[diff] - edge) <= 1e-9 * edge).all(), (b, h, int(diff.sum()))
                else:
                    assert abs(int(its[b, h]) - ref_it) <= 1, (its[b, h], ref_it)
                # threshold set, mass >= p, minimal up to ties
                thr = prob[mask].min()
                assert (prob[~mask] < thr).all() or not (~mask).any()
                assert prob[mask].sum() >= float(p) - 1e-12
                assert prob[prob > thr].sum() < float(p) + 1e-12
    sel_idx, sel_cnt = c.new_sel()
    c.topp_select_alg3(sc_dev, 1.0, sel_idx, sel_cnt)
    torch.cuda.synchronize()
    assert (sel_cnt.cpu().numpy() == n_seq[:, None]).all()
    c.close()


def test_topp_literal_config_tie_break(orc, rot128):
    """P9: literal BASELINE config 0 (sink keys = 2 x query): Top-p(0.9) = {0,1,2,3}, Top-p(0.7) = {0,1,2}."""
    import torch
    w = U.workload(0, variant="L")
    c = U.make_cache(w, rot128[0])
    c.encode_keys(U.to_dev(w.seq_lens))
    out = c.new_out()
    sel_idx, sel_cnt = c.new_sel()
    q = U.to_dev(w.q)
    for p, want in ((0.9, [0, 1, 2, 3]), (0.7, [0, 1, 2])):
        c.decode_step(q, p, out, sel_idx, sel_cnt)
        torch.cuda.synchronize()
        k = int(sel_cnt.cpu()[0, 0])
        assert sel_idx.cpu().numpy()[0, 0, :k].tolist() == want
    c.close()


# ---- S7: hybrid attention ------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg0", "cfg1_small", "cfg2_small", "cfg3_small"])
def test_sparse_attention_oracle_sets(orc, rot128, name):
    import torch
    w = get_case(name)
    o = U.oracle_full(orc, w, rot128[0])
    c = U.make_cache(w, rot128[0])
    U.load_index(c, o)
    out = c.new_out()
    lse = torch.zeros(w.B, w.Hq, device="cuda")
    c.sparse_attention(U.to_dev(w.q, U.torch_dtype(w)), U.to_dev(o["sel_idx"]), U.to_dev(o["sel_cnt"]), out, lse)
    torch.cuda.synchronize()
    U.assert_attention_close(out.cpu().numpy(), o["out"], w.kv_dtype)
    assert np.abs(out.cpu().numpy() - o["out"]).max() <= 1e-3 * max(1.0, np.abs(o["out"]).max())
    assert np.allclose(lse.cpu().numpy(), o["lse"], rtol=1e-4, atol=1e-3)
    c.close()


def test_sparse_attention_pending_window_and_empty(orc, rot128):
    """pending tokens [n_indexed, n_total) are always attended (L215); empty attended set -> 0 / -inf;
    bf16 output rounding."""
    import torch
    w = U.workload(3, L=1200, B=4)
    rng = np.random.default_rng(3)
    n_tot = w.seq_lens.copy()
    n_idx = np.maximum(0, n_tot - np.array([0, 37, 64, 5], np.int32)).astype(np.int32)
    n_idx[3] = 0
    n_tot[3] = 0                                        # sequence with nothing to attend
    sel_cnt = np.zeros((w.B, w.Hq), np.int32)
    sel_idx = np.zeros((w.B, w.Hq, w.Lcap), np.int32)
    for b in range(w.B):
        for h in range(w.Hq):
            k = 0 if n_idx[b] == 0 else int(rng.integers(0, min(600, n_idx[b])))
            if h == 1:
                k = 0                                   # only the pending window
            sel_cnt[b, h] = k
            sel_idx[b, h, :k] = rng.choice(max(1, n_idx[b]), k, replace=False)
    ref_out, ref_lse = orc.attention(w.q, w.K, w.V, sel_idx, sel_cnt, n_idx, n_tot, U.SM_SCALE)
    for out_dtype in (torch.float32, torch.bfloat16):
        c = U.make_cache(w, rot128[0], out_dtype=out_dtype)
        c.n_indexed.copy_(U.to_dev(n_idx))
        c.n_total.copy_(U.to_dev(n_tot))
        out = c.new_out()
        lse = torch.zeros(w.B, w.Hq, device="cuda")
        c.sparse_attention(U.to_dev(w.q, torch.bfloat16), U.to_dev(sel_idx), U.to_dev(sel_cnt), out, lse)
        torch.cuda.synchronize()
        got = out.float().cpu().numpy()
        U.assert_attention_close(got, ref_out, "bf16")
        assert (got[3] == 0).all() and np.isneginf(lse.cpu().numpy()[3]).all()
        assert np.allclose(lse.cpu().numpy()[:3], ref_lse[:3], rtol=1e-4, atol=1e-3)
        c.close()
