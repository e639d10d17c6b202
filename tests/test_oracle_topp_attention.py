"""Pins for oracle O6 (adaptive Top-p), O7 (hybrid attention), O8 (lazy updates).  CPU only.

P5  the Top-p set is the minimal set whose estimated mass is >= p:
    ordering property, mass property, minimality, brute force over all subsets for tiny rows,
    cross-check against the paper's own Alg.3 (L217-252, restored `else`).
P9  literal BASELINE config 0 (sink keys = 2 x query): Top-p(0.9) = {0,1,2,3}, Top-p(0.7) =
    {0,1,2} by the lowest-index tie-break.
P6  p = 1 reproduces dense softmax attention (textbook definition, numpy and torch SDPA).
"""
import itertools
import math

import numpy as np
import pytest

from paper_2606_31519_b200 import synth

D = 128


def softmax64(s):
    w = np.exp(s.astype(np.float64) - s.astype(np.float64).max())
    return w / w.sum()


def check_topp_properties(scores, sel, p, slack=0.0):
    """(i) every selected prob >= every unselected (tie => lower index selected);
    (ii) mass(sel) >= p; (iii) mass(sel) - min selected prob < p."""
    pr = softmax64(scores)
    sel = np.asarray(sel)
    assert len(set(sel.tolist())) == len(sel)
    mask = np.zeros(len(scores), bool)
    mask[sel] = True
    if mask.all():
        return
    pmin_sel = pr[mask].min()
    pmax_uns = pr[~mask].max()
    assert pmin_sel >= pmax_uns - slack
    if slack == 0.0:
        ties_sel = np.where(mask & (pr == pmax_uns))[0]
        ties_uns = np.where(~mask & (pr == pmax_uns))[0]
        if len(ties_sel) and len(ties_uns):
            assert ties_sel.max() < ties_uns.min()
    mass = pr[mask].sum()
    assert mass >= p - 1e-12 - slack
    assert mass - pmin_sel < p + 1e-12 + slack


def test_p5_properties_random_rows(orc):
    rng = np.random.default_rng(4)
    rows, L = 12, 3000
    scores = (rng.standard_normal((rows, L)) * rng.uniform(0.5, 6, (rows, 1))).astype(np.float32)
    scores[3, :50] = scores[3, 0]           # a block of exact ties
    scores[4] = 1.25                         # all equal
    n = np.full(rows, L, np.int32)
    n[5] = 1
    n[6] = 0
    n[7] = 777
    for p in (0.5, 0.9, 0.95, 0.999):
        idx, cnt = orc.topp(scores, n, p)
        for r in range(rows):
            if n[r] == 0:
                assert cnt[r] == 0
                continue
            sel = idx[r, :cnt[r]]
            assert sel.max() < n[r]
            check_topp_properties(scores[r, :n[r]], sel, p)
        assert cnt[4] == math.ceil(p * L - 1e-9) and (np.sort(idx[4, :cnt[4]]) == np.arange(cnt[4])).all()
        assert cnt[5] == 1


def test_p5_bruteforce_minimal_subset(orc):
    rng = np.random.default_rng(9)
    for trial in range(40):
        L = int(rng.integers(2, 12))
        s = (rng.standard_normal(L) * 2).astype(np.float32)
        if trial % 5 == 0:
            s[: L // 2] = s[0]
        p = float(rng.uniform(0.3, 0.98))
        idx, cnt = orc.topp(s[None], [L], p)
        pr = softmax64(s)
        best = None
        for k in range(1, L + 1):
            if any(pr[list(c)].sum() >= p for c in itertools.combinations(range(L), k)):
                best = k
                break
        assert cnt[0] == best
        check_topp_properties(s, idx[0, :cnt[0]], p)


def test_p5_alg3_crosscheck(orc):
    rng = np.random.default_rng(21)
    for trial in range(30):
        L = int(rng.integers(50, 4000))
        s = (rng.standard_normal(L) * rng.uniform(1, 5)).astype(np.float32)
        if trial % 4 == 0:
            s[10:20] = s[10]
        p = float(rng.choice([0.65, 0.8, 0.9, 0.95]))
        pr = softmax64(s)
        mask, iters = orc.topp_alg3(pr, p)
        assert 0 < iters < 200
        idx, cnt = orc.topp(s[None], [L], p)
        sel = np.zeros(L, bool)
        sel[idx[0, :cnt[0]]] = True
        boundary = pr[sel].min()
        # Alg.3 returns S > theta: every entry >= the boundary value (all ties included)
        assert (mask == (pr >= boundary)).all()
        assert (mask | ~sel).all()
        if (pr == boundary).sum() == 1:
            assert (mask == sel).all()


def test_p_ge_1_selects_everything(orc):
    s = np.random.default_rng(1).standard_normal((2, 100)).astype(np.float32)
    idx, cnt = orc.topp(s, [100, 60], 1.0)
    assert cnt.tolist() == [100, 60]
    assert (np.sort(idx[1, :60]) == np.arange(60)).all()


def test_p9_literal_config0_sinks(orc, rot128):
    r32, _ = rot128
    w = synth.make_workload(0, variant="L")
    ck = orc.centroid(w.K, w.seq_lens)
    codes, fs, fb = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck)
    assert (codes[0, 0, 0] == codes[0, 0, 1]).all() and fs[0, 0, 0] == fs[0, 0, 3]
    sm = 1 / math.sqrt(D)
    res = orc.decode_step(w.q, w.K, w.V, codes, fs, fb, ck, None, w.seq_lens, w.seq_lens, 0, r32, 0.9, sm)
    assert sorted(res["sel_idx"][0, 0, :res["sel_cnt"][0, 0]].tolist()) == [0, 1, 2, 3]
    s = res["scores"][0, 0]
    assert s[0] == s[1] == s[2] == s[3] and s[0] > s[4:4096].max() + 50
    res7 = orc.decode_step(w.q, w.K, w.V, codes, fs, fb, ck, None, w.seq_lens, w.seq_lens, 0, r32, 0.7, sm)
    assert res7["sel_idx"][0, 0, :res7["sel_cnt"][0, 0]].tolist() == [0, 1, 2]


def _dense_attention(q, K, V, n, sm):
    l = (K[:n].astype(np.float64) @ q.astype(np.float64)) * sm
    w = np.exp(l - l.max())
    return (w / w.sum()) @ V[:n].astype(np.float64), l.max() + math.log(w.sum())


def test_p6_p1_is_dense_attention(orc, rot128):
    import torch
    r32, _ = rot128
    w = synth.make_workload(1, L=600 + 11)
    L = int(w.seq_lens[0])
    ck = orc.centroid(w.K, w.seq_lens)
    codes, fs, fb = orc.encode(w.K, [0], w.seq_lens, 0, r32, ck)
    sm = 1 / math.sqrt(D)
    res = orc.decode_step(w.q, w.K, w.V, codes, fs, fb, ck, None, w.seq_lens, w.seq_lens, 0, r32, 1.0, sm)
    assert (res["sel_cnt"] == L).all()
    for h in range(w.Hq):
        ref, lse = _dense_attention(w.q[0, h], w.K[0, h // w.G], w.V[0, h // w.G], L, sm)
        np.testing.assert_allclose(res["out"][0, h], ref, rtol=1e-5, atol=1e-5)
        assert res["lse"][0, h] == pytest.approx(lse, rel=1e-6)
    # library routine: torch SDPA on CPU in fp64 with GQA expansion
    qt = torch.from_numpy(w.q.astype(np.float64))[:, :, None, :]                     # [1,Hq,1,D]
    Kt = torch.from_numpy(w.K[:, :, :L].astype(np.float64)).repeat_interleave(w.G, dim=1)
    Vt = torch.from_numpy(w.V[:, :, :L].astype(np.float64)).repeat_interleave(w.G, dim=1)
    o = torch.nn.functional.scaled_dot_product_attention(qt, Kt, Vt, scale=sm)[:, :, 0].numpy()
    np.testing.assert_allclose(res["out"], o, rtol=1e-5, atol=1e-5)


def test_o7_subset_and_pending_and_empty(orc):
    rng = np.random.default_rng(6)
    B, Hq, Hkv, Lcap = 2, 4, 2, 64
    q = rng.standard_normal((B, Hq, D)).astype(np.float32)
    K = rng.standard_normal((B, Hkv, Lcap, D)).astype(np.float32)
    V = rng.standard_normal((B, Hkv, Lcap, D)).astype(np.float32)
    sel_idx = np.zeros((B, Hq, Lcap), np.int32)
    sel_cnt = np.zeros((B, Hq), np.int32)
    sel_idx[0, 0, :3] = [5, 1, 9]
    sel_cnt[0, 0] = 3
    sel_cnt[0, 1] = 0
    n_idx = np.array([40, 0], np.int32)
    n_tot = np.array([44, 0], np.int32)
    sm = 0.3
    out, lse = orc.attention(q, K, V, sel_idx, sel_cnt, n_idx, n_tot, sm)
    for h, toks in ((0, [5, 1, 9, 40, 41, 42, 43]), (1, [40, 41, 42, 43])):
        l = (K[0, h // 2, toks].astype(np.float64) @ q[0, h].astype(np.float64)) * sm
        wgt = np.exp(l - l.max())
        np.testing.assert_allclose(out[0, h], (wgt / wgt.sum()) @ V[0, h // 2, toks].astype(np.float64),
                                   rtol=1e-6, atol=1e-6)
    assert (out[1] == 0).all() and np.isneginf(lse[1]).all()      # empty attended set


def test_o8_lazy_index_state_machine(orc, rot128):
    r32, _ = rot128
    w = synth.make_workload(3, L=256, B=2, extra_cap=32)
    W = 8
    st = orc.LazyIndex(w.K, w.V, w.seq_lens, 0, r32, W)
    n0 = w.seq_lens.copy()
    ck0 = st.c_k.copy()
    for step in range(1, 20):
        kn, vn = synth.append_rows(3, step, 2, w.Hkv, 1)
        st.append(kn, vn)
        assert (st.n_total == n0 + step).all()
        pend = st.n_total - st.n_indexed
        assert (pend <= W).all() and (pend >= 1).all()
        # committed one call after the flush was enqueued (R14)
        assert (st.n_indexed == n0 + ((step - 1) // W) * W).all()
        assert st.in_flight == (W if step % W == 0 else 0)
        assert (st.c_k == ck0).all()                   # centroid frozen
    # flushed codes equal a direct encode of the same rows with the frozen centroid
    c_ref, f_ref, _ = orc.encode(st.K, n0, n0 + 16, 0, r32, ck0)
    for b in range(2):
        sl = slice(int(n0[b]), int(n0[b]) + 16)
        assert (st.codes[b, :, sl] == c_ref[b, :, sl]).all() and (st.f_scale[b, :, sl] == f_ref[b, :, sl]).all()
        assert (st.codes[b, :, int(n0[b]) + 16:] == 0).all()
