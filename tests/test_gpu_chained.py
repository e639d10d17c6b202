"""Chained GPU parity: the whole path on the GPU (encode -> query -> estimate -> Top-p -> attention,
and the fused rbq_decode_step), against the oracle end to end; p = 1 against dense attention (P6);
lazy append / flush state machine (L215) against the oracle's LazyIndex, with and without a side stream.

In the chained runs the GPU's own fp32 logits feed its Top-p, so a set difference is additionally
allowed for tokens whose logit lies within the 1e-5 band of the boundary logit: the check used here is
"oracle Top-p applied to the GPU's logits" (exact rule) plus the end-to-end output tolerance.
"""
import numpy as np
import pytest

from tests import gpu_util as U

pytestmark = pytest.mark.gpu

ROT_DENSE, ROT_WH = 0, 1


def _chained(orc, w, rot, kind, p, with_cq=False, factor_f16=False):
    import torch
    o = U.oracle_full(orc, w, rot, kind, with_cq, p=p, factor_f16=factor_f16)
    c = U.make_cache(w, rot, rot_kind=kind, with_cq=with_cq, **(dict(factor_dtype=torch.float16) if factor_f16 else {}))
    c.encode_keys(U.to_dev(w.seq_lens))
    q = U.to_dev(w.q, U.torch_dtype(w))
    # staged calls
    scores = c.new_scores()
    sel_idx, sel_cnt = c.new_sel()
    out, out2 = c.new_out(), c.new_out()
    c.estimate_scores(q, scores)
    c.topp_select(scores, p, sel_idx, sel_cnt)
    c.sparse_attention(q, sel_idx, sel_cnt, out)
    # fused call
    sel_idx2, sel_cnt2 = c.new_sel()
    c.decode_step(q, p, out2, sel_idx2, sel_cnt2)
    # fused call without index lists: the selection stays a bitmap in the workspace
    out3, sel_cnt3 = c.new_out(), c.new_sel()[1]
    c.decode_step(q, p, out3, None, sel_cnt3)
    torch.cuda.synchronize()
    U.assert_same_step_output(out3.cpu().numpy(), out2.cpu().numpy(), "fused without lists != fused")
    assert (sel_cnt3.cpu().numpy() == sel_cnt2.cpu().numpy()).all()
    s = scores.cpu().numpy()
    U.assert_logits_close(s, o["scores"], w.seq_lens, w.Hq)
    idx, cnt = sel_idx.cpu().numpy(), sel_cnt.cpu().numpy()
    assert (cnt == sel_cnt2.cpu().numpy()).all()
    n_rows = np.repeat(w.seq_lens, w.Hq)
    ref_idx, ref_cnt = orc.topp(s.reshape(w.B * w.Hq, w.Lcap), n_rows, p)     # exact rule on the GPU's logits
    ref_idx, ref_cnt = ref_idx.reshape(w.B, w.Hq, w.Lcap), ref_cnt.reshape(w.B, w.Hq)
    idx2 = sel_idx2.cpu().numpy()
    for b in range(w.B):
        n = int(w.seq_lens[b])
        for h in range(w.Hq):
            g = idx[b, h, :cnt[b, h]]
            assert (g == idx2[b, h, :cnt[b, h]]).all(), "fused and staged selections differ"
            U.assert_topp_row(s[b, h, :n], g, ref_idx[b, h, :ref_cnt[b, h]], p)
    # budgets of the oracle chain and the GPU chain agree closely (boundary tokens only)
    assert np.abs(cnt.astype(np.int64) - o["sel_cnt"]).max() <= max(2, int(0.002 * o["sel_cnt"].max()))
    U.assert_attention_close(out.cpu().numpy(), o["out"], w.kv_dtype)
    U.assert_same_step_output(out.cpu().numpy(), out2.cpu().numpy(), "fused != staged output")
    c.close()
    return o


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("cfg,kw,p", [(0, {}, 0.9), (1, dict(L=5003), 0.8), (1, dict(L=5003), 0.95),
                                      (2, dict(L=6150, n_heavy=32), 0.9), (3, dict(L=3001, B=3), 0.9)])
def test_decode_step_chained(orc, rot128, cfg, kw, p, kind):
    from paper_2606_31519_b200 import synth
    rot = rot128[0] if kind == ROT_DENSE else synth.wh_sign_vector(128)
    _chained(orc, U.workload(cfg, **kw), rot, kind, p)


@pytest.mark.parametrize("force", ["0", "1"])
@pytest.mark.parametrize("cfg,kw,p", [(1, dict(L=5003), 0.9), (3, dict(L=3001, B=7), 0.9), (3, dict(L=2500, B=24), 0.8),
                                      (4, dict(L=4099, B=2), 0.95),
                                      (1, dict(L=3001, Hq=8, Hkv=8), 0.9),      # G = 1: one bitmap row per group
                                      (1, dict(L=4100, Hq=12, Hkv=6), 0.9),     # G = 2
                                      (3, dict(L=1500, B=5, Hq=4, Hkv=1), 0.8),
                                      (1, dict(L=70, Hq=4, Hkv=2), 0.6),        # fewer attended rows than CTAs
                                      (1, dict(L=33, n_heavy=4), 0.9)])         # two bitmap words, the second with one token
def test_decode_step_chained_both_gather_paths(orc, rot128, cfg, kw, p, force, monkeypatch):
    """S7 has two paths for bf16 K/V: straight from the selection bitmaps (dynamic hand-out of a group's bitmap words, work
    partition by estimated union sizes; the default) and through attn_plan_kernel + union lists (RBQ_GATHER_PLAN=1).  Both
    are forced here on shapes with one, a few and many KV groups per CTA (ranges that straddle several groups, groups shared
    by several CTAs, whole groups inside one CTA's range) and run through the whole chain against the oracle."""
    monkeypatch.setenv("RBQ_GATHER_PLAN", force)
    _chained(orc, U.workload(cfg, **kw), rot128[0], ROT_DENSE, p)


def test_plan_path_is_bit_reproducible_and_matches_default(rot128, monkeypatch):
    """RBQ_GATHER_PLAN=1 (static partition over union lists) gives the same bits on every run; the default path (dynamic
    hand-out) agrees with it to the accumulation-order bound, run after run, also while its union-size history (rho) settles
    over the first steps and after the query has changed."""
    import torch
    from paper_2606_31519_b200 import synth
    w = U.workload(2, L=9000, n_heavy=32)
    pool = synth.query_pool(w, 3)
    outs = {}
    for force in ("1", "0"):
        monkeypatch.setenv("RBQ_GATHER_PLAN", force)
        c = U.make_cache(w, rot128[0])
        c.encode_keys(U.to_dev(w.seq_lens))
        res = []
        for i in range(6):
            q = U.to_dev(pool[i % 3], U.torch_dtype(w))
            o = c.new_out()
            c.decode_step(q, 0.9, o)
            torch.cuda.synchronize()
            res.append(o.cpu().numpy())
        outs[force] = res
        c.close()
    for i in range(3):                                    # same query three steps later: same bits on the static path
        assert (outs["1"][i].view(np.uint32) == outs["1"][i + 3].view(np.uint32)).all()
    for i in range(6):
        U.assert_same_step_output(outs["0"][i], outs["1"][i], f"default path differs from the plan path at step {i}")


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("cfg,kw,D", [(1, dict(L=5003), 128), (3, dict(L=3001, B=3), 128), (1, dict(L=3001), 64), (2, dict(L=4100, n_heavy=32), 256)])
def test_decode_step_chained_f16_factors(orc, cfg, kw, D, kind):
    """2-byte correction factors: rbq_config.factor_dtype = RBQ_F16.  The stored
    factors are the oracle's fp32 factors rounded to binary16 bit for bit; logits, Top-p sets and outputs then match the
    oracle run on those rounded factors at the usual tolerances (the rounding itself moves a logit by <= 2^-11 of its
    estimated part: tests/test_oracle_rotation_encode.py::test_factors_f16_rounding_and_logit_bound)."""
    import torch
    w = U.workload(cfg, D=D, **kw)
    rot = U.rotation(orc, D, kind)
    o = _chained(orc, w, rot, kind, 0.9, factor_f16=True)
    c = U.make_cache(w, rot, rot_kind=kind, factor_dtype=torch.float16)
    c.encode_keys(U.to_dev(w.seq_lens))
    torch.cuda.synchronize()
    fs = c.f_scale.cpu().numpy()
    assert fs.dtype == np.float16
    for b in range(w.B):
        n = int(w.seq_lens[b])
        assert (fs[b, :, :n].view(np.uint16) == o["f_scale"][b, :, :n].astype(np.float16).view(np.uint16)).all(), "fp16 factors differ"
        assert (c.codes.cpu().numpy().view(np.uint32)[b, :, :n] == o["codes"][b, :, :n]).all()
    c.close()


def test_back_to_back_steps_with_different_queries(orc, rot128):
    """Six decode steps enqueued back to back without a host synchronize, each with its own q and its own output buffer:
    S3 of step n + 1 is launched with programmatic stream serialisation and may become resident under the tail of step
    n's gather attention, so it must neither overwrite the query constants step n still reads nor read q early.  Every
    step's output, budgets and selected sets against the oracle; then the same six queries again in reverse order."""
    import torch
    from paper_2606_31519_b200 import synth
    w = U.workload(1, L=9001)
    rot = rot128[0]
    o = U.oracle_index(orc, w, rot, ROT_DENSE)
    c = U.make_cache(w, rot)
    c.encode_keys(U.to_dev(w.seq_lens))
    pool = synth.query_pool(w, 6)
    dt = U.torch_dtype(w)
    q_dev = [U.to_dev(pool[i], dt) for i in range(6)]
    refs = [orc.decode_step(pool[i], w.K, w.V, o["codes"], o["f_scale"], None, o["c_k"], None, o["n_indexed"], o["n_total"],
                            ROT_DENSE, rot, w.p, U.SM_SCALE) for i in range(6)]
    for order in (range(6), reversed(range(6))):
        order = list(order)
        outs = [c.new_out() for _ in order]
        cnts = [c.new_sel()[1] for _ in order]
        for k, i in enumerate(order):
            c.decode_step(q_dev[i], w.p, outs[k], None, cnts[k])
        torch.cuda.synchronize()
        for k, i in enumerate(order):
            U.assert_attention_close(outs[k].cpu().numpy(), refs[i]["out"], w.kv_dtype)
            d = np.abs(cnts[k].cpu().numpy().astype(np.int64) - refs[i]["sel_cnt"])
            assert d.max() <= max(2, int(0.002 * refs[i]["sel_cnt"].max())), f"step {k} (query {i}): budgets differ by {d.max()}"
    c.close()


def test_decode_step_chained_with_cq(orc, rot128):
    _chained(orc, U.workload(0, with_cq=True), rot128[0], ROT_DENSE, 0.9, with_cq=True)


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(L=2051)), (3, dict(L=1500, B=3))])
def test_p1_is_dense_attention(orc, rot128, cfg, kw):
    """P6: rbq_decode_step(p = 1) == textbook softmax attention over all tokens (oracle with the full index
    set, and torch SDPA in fp32 on the same device as an independent library definition)."""
    import torch
    w = U.workload(cfg, **kw)
    c = U.make_cache(w, rot128[0])
    c.encode_keys(U.to_dev(w.seq_lens))
    q = U.to_dev(w.q, U.torch_dtype(w))
    out = c.new_out()
    sel_idx, sel_cnt = c.new_sel()
    c.decode_step(q, 1.0, out, sel_idx, sel_cnt)
    torch.cuda.synchronize()
    assert (sel_cnt.cpu().numpy() == w.seq_lens[:, None]).all()
    all_idx = np.broadcast_to(np.arange(w.Lcap, dtype=np.int32), (w.B, w.Hq, w.Lcap)).copy()
    all_cnt = np.broadcast_to(w.seq_lens[:, None], (w.B, w.Hq)).astype(np.int32).copy()
    ref, _ = orc.attention(w.q, w.K, w.V, all_idx, all_cnt, w.seq_lens, w.seq_lens, U.SM_SCALE)
    U.assert_attention_close(out.cpu().numpy(), ref, w.kv_dtype)
    G = w.Hq // w.Hkv
    for b in range(w.B):
        n = int(w.seq_lens[b])
        kk = c.K[b, :, :n].float().repeat_interleave(G, dim=0)
        vv = c.V[b, :, :n].float().repeat_interleave(G, dim=0)
        sd = torch.nn.functional.scaled_dot_product_attention(q[b].float()[:, None, :], kk, vv)[:, 0]
        U.assert_attention_close(out[b].cpu().numpy(), sd.cpu().numpy(), w.kv_dtype)
    c.close()


@pytest.mark.parametrize("use_side", [False, True])
@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
def test_append_flush_state_machine(orc, rot128, use_side, kind):
    """L215 lazy updates (R14): 1 token per step, W = 8; flush enqueued when pending reaches W, committed by
    the next append; codes of flushed rows bit-exact, decode output checked at steps around each flush."""
    import torch
    from paper_2606_31519_b200 import synth
    W, steps = 8, 21
    w = U.workload(3, L=900, B=3, extra_cap=64)
    rot = rot128[0] if kind == ROT_DENSE else synth.wh_sign_vector(128)
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, kind, rot, W)
    c = U.make_cache(w, rot, rot_kind=kind, flush_tokens=W)
    c.encode_keys(U.to_dev(w.seq_lens))
    main = torch.cuda.current_stream()
    side = torch.cuda.Stream() if use_side else None
    pool = synth.query_pool(w, 4)
    out = c.new_out()
    sel_idx, sel_cnt = c.new_sel()
    for s in range(steps):
        k_new, v_new = synth.append_rows(3, s, w.B, w.Hkv, 1)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16), stream=main, side_stream=side)
        q_np = pool[s % 4]
        c.decode_step(U.to_dev(q_np, torch.bfloat16), 0.9, out, sel_idx, sel_cnt)
        torch.cuda.synchronize()
        assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all(), f"step {s}: n_indexed"
        assert (c.n_total.cpu().numpy() == lazy.n_total).all(), f"step {s}: n_total"
        if s in (0, W - 2, W - 1, W, W + 1, 2 * W - 1, 2 * W, steps - 1):
            ref = orc.decode_step(q_np, lazy.K, lazy.V, lazy.codes, lazy.f_scale, None, lazy.c_k, None, lazy.n_indexed,
                                  lazy.n_total, kind, rot, 0.9, U.SM_SCALE)
            U.assert_attention_close(out.cpu().numpy(), ref["out"], "bf16")
            assert np.abs(sel_cnt.cpu().numpy().astype(np.int64) - ref["sel_cnt"]).max() <= 2
    # every committed or in-flight row carries the oracle's code and factor; K/V rows were copied verbatim
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    for b in range(w.B):
        n = int(lazy.n_indexed[b]) + lazy.in_flight
        assert (codes[b, :, :n] == lazy.codes[b, :, :n]).all()
        assert (fs[b, :, :n].view(np.uint32) == lazy.f_scale[b, :, :n].view(np.uint32)).all()
        nt = int(lazy.n_total[b])
        assert (c.K[b, :, :nt].float().cpu().numpy() == lazy.K[b, :, :nt]).all()
        assert (c.V[b, :, :nt].float().cpu().numpy() == lazy.V[b, :, :nt]).all()
    c.close()


@pytest.mark.parametrize("force", ["0", "1"])
def test_large_pending_window_both_gather_paths(orc, rot128, force, monkeypatch):
    """A pending window of several hundred rows (W = 1024: nothing is flushed), appended 100 / 200 / 61 rows at a time: the
    pending rows follow the bitmap words of a KV group as many words of 32 rows, claims straddle the border between the two,
    the last pending word is ragged.  Output against the oracle's step after each append, on both S7 paths."""
    import torch
    from paper_2606_31519_b200 import synth
    monkeypatch.setenv("RBQ_GATHER_PLAN", force)
    W = 1024
    w = U.workload(3, L=1700, B=3, extra_cap=512)
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, ROT_DENSE, rot128[0], W)
    c = U.make_cache(w, rot128[0], flush_tokens=W)
    c.encode_keys(U.to_dev(w.seq_lens))
    pool = synth.query_pool(w, 3)
    out = c.new_out()
    for s, n_new in enumerate((100, 200, 61)):
        k_new, v_new = synth.append_rows(3, 40 + s, w.B, w.Hkv, n_new)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16))
        c.decode_step(U.to_dev(pool[s], torch.bfloat16), 0.9, out)
        torch.cuda.synchronize()
        assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all() and (c.n_total.cpu().numpy() == lazy.n_total).all()
        assert int((lazy.n_total - lazy.n_indexed).min()) == sum((100, 200, 61)[:s + 1])
        ref = orc.decode_step(pool[s], lazy.K, lazy.V, lazy.codes, lazy.f_scale, None, lazy.c_k, None, lazy.n_indexed,
                              lazy.n_total, ROT_DENSE, rot128[0], 0.9, U.SM_SCALE)
        U.assert_attention_close(out.cpu().numpy(), ref["out"], "bf16")
    c.close()


def test_append_flush_enc_fast(orc, rot128):
    """Lazy flush through RBQ_ENC_FAST (tcgen05 encode with per-sequence t_begin / t_count, tiles far from full): the
    flushed rows carry the oracle's codes up to the guard band (|y_j| <= 1e-5 ||x||) and its factors within 1e-5."""
    import torch
    from paper_2606_31519_b200 import binding as rb, synth
    W = 64
    w = U.workload(3, L=1500, B=3, extra_cap=256)
    rot = rot128[0]
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, ROT_DENSE, rot, W)
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, torch.from_numpy(rot), flush_tokens=W, enc_mode=rb.RBQ_ENC_FAST)
    c.K.copy_(U.to_dev(w.K, torch.bfloat16))
    c.V.copy_(U.to_dev(w.V, torch.bfloat16))
    c.encode_keys(U.to_dev(w.seq_lens))
    side = torch.cuda.Stream()
    for s, n_new in enumerate([40, 40, 64, 30, 100]):
        k_new, v_new = synth.append_rows(3, 90 + s, w.B, w.Hkv, n_new)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16), side_stream=side)
        torch.cuda.synchronize()
        assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all() and (c.n_total.cpu().numpy() == lazy.n_total).all()
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    P = rot.astype(np.float64)
    n0 = w.seq_lens
    for b in range(w.B):
        n = int(lazy.n_indexed[b]) + lazy.in_flight
        assert n > int(n0[b])
        for g in range(w.Hkv):
            x = lazy.K[b, g, :n].astype(np.float64) - lazy.c_k[b, g].astype(np.float64)
            y = x @ P
            xn = np.linalg.norm(x, axis=1, keepdims=True)
            diff = codes[b, g, :n] ^ lazy.codes[b, g, :n]
            bits = ((diff[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(n, 128).astype(bool)
            assert (np.abs(y)[bits] <= 1e-5 * np.broadcast_to(xn, y.shape)[bits]).all()
            ref = lazy.f_scale[b, g, :n].astype(np.float64)
            assert (np.abs(fs[b, g, :n] - ref) <= 1e-5 * np.abs(ref)).all()
    c.close()


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
def test_encode_fast_with_cq(orc, rot128, kind):
    """RBQ_ENC_FAST with a query centroid: f_bias = <c_q, k> must be written by rbq_encode_keys AND by
    the lazy flush in the tensor-core encode mode too, bit-identical to the oracle's canonical chain (it does not go
    through the rotation); the logits of the fused path then carry the Eq.2 term <c_q, k>."""
    import torch
    from paper_2606_31519_b200 import binding as rb, synth
    W = 64
    w = U.workload(1, L=3001, with_cq=True, extra_cap=192)
    rot = rot128[0] if kind == ROT_DENSE else synth.wh_sign_vector(128)
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, kind, rot, W, c_q=w.c_q)
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)), flush_tokens=W,
                       rot_kind=kind, enc_mode=rb.RBQ_ENC_FAST, with_cq=True)
    c.K.copy_(U.to_dev(w.K, torch.bfloat16))
    c.V.copy_(U.to_dev(w.V, torch.bfloat16))
    c.c_q.copy_(U.to_dev(w.c_q))
    c.f_bias.fill_(float("nan"))
    c.encode_keys(U.to_dev(w.seq_lens))
    for s_, n_new in enumerate([70, 60]):                        # two flushes (64 rows each), the second commits the first
        k_new, v_new = synth.append_rows(1, 300 + s_, w.B, w.Hkv, n_new)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16))
    torch.cuda.synchronize()
    fb = c.f_bias.cpu().numpy()
    n = int(lazy.n_indexed[0]) + lazy.in_flight
    assert n == 3001 + 128
    assert (fb[0, :, :n].view(np.uint32) == lazy.f_bias[0, :, :n].view(np.uint32)).all(), "f_bias differs in RBQ_ENC_FAST"
    # logits through the GPU's own (guard-band) index: compare with the oracle's logits on the GPU's codes / factors
    scores = c.new_scores()
    q = U.to_dev(w.q, torch.bfloat16)
    c.estimate_scores(q, scores)
    torch.cuda.synchronize()
    ni = c.n_indexed.cpu().numpy()
    ref, _, _, _ = orc.estimate_scores(w.q, c.codes.cpu().numpy().view(np.uint32), c.f_scale.cpu().numpy(), fb, c.c_k.cpu().numpy(),
                                       w.c_q, ni, kind, rot, U.SM_SCALE)
    U.assert_logits_close(scores.cpu().numpy(), ref, ni, w.Hq)
    c.close()


def test_append_beyond_capacity_is_dropped_and_flagged(orc, rot128):
    """Appending past max_tokens: the extra rows are dropped, n_total is clamped to Lcap, the sticky status bit is
    set, nothing outside the sequence's own cache rows is touched, and a decode step still runs on the clamped state."""
    import torch
    from paper_2606_31519_b200 import synth
    w = U.workload(3, L=500, B=2)                       # Lcap = 512 (seq_lens <= 500)
    c = U.make_cache(w, rot128[0], flush_tokens=8)
    c.encode_keys(U.to_dev(w.seq_lens))
    assert c.status_flags() == 0
    guard_k = c.K.clone()
    room = int(w.Lcap - w.seq_lens.max())
    k_new, v_new = synth.append_rows(3, 7, w.B, w.Hkv, room + 24)
    c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16))
    out = c.new_out()
    c.decode_step(U.to_dev(w.q, torch.bfloat16), 0.9, out)
    torch.cuda.synchronize()
    assert c.status_flags() == 1
    nt = c.n_total.cpu().numpy()
    assert (nt <= w.Lcap).all() and nt.max() == w.Lcap and (c.n_indexed.cpu().numpy() <= nt).all()
    for b in range(w.B):
        n0 = int(w.seq_lens[b])
        m = int(nt[b]) - n0
        assert (c.K[b, :, :n0] == guard_k[b, :, :n0]).all(), "old rows were overwritten"
        assert (c.K[b, :, n0:n0 + m].float().cpu().numpy() == k_new[b, :, :m]).all()
    assert torch.isfinite(out).all()
    c.append_tokens(U.to_dev(k_new[:, :, :8], torch.bfloat16), U.to_dev(v_new[:, :, :8], torch.bfloat16))   # commits the flush
    torch.cuda.synchronize()
    assert (c.n_indexed.cpu().numpy() <= c.n_total.cpu().numpy()).all() and (c.n_total.cpu().numpy() <= w.Lcap).all()
    c.close()


@pytest.mark.parametrize("fast", [False, True])
def test_pipelined_prefill_side_stream(orc, rot128, fast):
    """Asynchronous pipelined prefill ("a secondary, low-priority CUDA stream ... the quantization process
    proceeds in parallel with the heavy attention computation", L341 "<10 % TTFT overhead"): rbq_encode_keys
    (centroid + Alg.1) runs on a low-priority stream while a dense causal attention of the same layer (torch SDPA, a
    library call standing in for the model) occupies the main stream; the two are joined by an event before the first
    decode step.  The index built under that contention must be the oracle's (bit for bit in RBQ_ENC_EXACT, inside the
    guard band in RBQ_ENC_FAST), and the decode step that follows must see it."""
    import torch
    from paper_2606_31519_b200 import binding as rb
    w = U.workload(1, L=16384)
    rot = rot128[0]
    o = U.oracle_full(orc, w, rot)
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, torch.from_numpy(rot), enc_mode=rb.RBQ_ENC_FAST if fast else rb.RBQ_ENC_EXACT)
    c.K.copy_(U.to_dev(w.K, torch.bfloat16))
    c.V.copy_(U.to_dev(w.V, torch.bfloat16))
    seq = U.to_dev(w.seq_lens)
    n = int(w.seq_lens[0])
    G = w.Hq // w.Hkv
    qs = torch.randn(1, w.Hq, n, 128, device="cuda", dtype=torch.bfloat16)          # the prefill's own queries
    kk = c.K[:, :, :n].repeat_interleave(G, dim=1).contiguous()
    vv = c.V[:, :, :n].repeat_interleave(G, dim=1).contiguous()
    lo, hi = torch.cuda.Stream.priority_range()
    main, side = torch.cuda.current_stream(), torch.cuda.Stream(priority=lo)
    torch.cuda.synchronize()
    side.wait_stream(main)
    for _ in range(2):                                                               # attention in flight on the main stream ...
        att = torch.nn.functional.scaled_dot_product_attention(qs, kk, vv, is_causal=True)
    c.encode_keys(seq, stream=side)                                                  # ... index build beside it
    done = torch.cuda.Event()
    done.record(side)
    main.wait_event(done)                                                            # "until the first decoding step of that layer"
    out = c.new_out()
    sel_cnt = c.new_sel()[1]
    c.decode_step(U.to_dev(w.q, torch.bfloat16), w.p, out, None, sel_cnt)
    torch.cuda.synchronize()
    assert torch.isfinite(att).all()
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    if not fast:
        assert (codes[0, :, :n] == o["codes"][0, :, :n]).all() and (fs[0, :, :n].view(np.uint32) == o["f_scale"][0, :, :n].view(np.uint32)).all()
        U.assert_attention_close(out.cpu().numpy(), o["out"], "bf16")
        assert np.abs(sel_cnt.cpu().numpy().astype(np.int64) - o["sel_cnt"]).max() <= max(2, int(0.002 * o["sel_cnt"].max()))
    else:
        P = rot.astype(np.float64)
        for g in range(w.Hkv):
            x = w.K[0, g, :n].astype(np.float64) - o["c_k"][0, g].astype(np.float64)
            y = x @ P
            xn = np.linalg.norm(x, axis=1, keepdims=True)
            diff = codes[0, g, :n] ^ o["codes"][0, g, :n]
            bits = ((diff[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(n, 128).astype(bool)
            assert (np.abs(y)[bits] <= 1e-5 * np.broadcast_to(xn, y.shape)[bits]).all()
            ref = o["f_scale"][0, g, :n].astype(np.float64)
            assert (np.abs(fs[0, g, :n] - ref) <= 1e-5 * np.abs(ref)).all()
        U.assert_attention_close(out.cpu().numpy(), o["out"], "bf16")
    c.close()


def test_append_many_tokens_per_call(orc, rot128):
    """n_new = 5 per call with W = 8 (flush of whole windows only), and n_new >= W in one call."""
    import torch
    from paper_2606_31519_b200 import synth
    W = 8
    w = U.workload(3, L=700, B=2, extra_cap=128)
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, ROT_DENSE, rot128[0], W)
    c = U.make_cache(w, rot128[0], flush_tokens=W)
    c.encode_keys(U.to_dev(w.seq_lens))
    out = c.new_out()
    for s, n_new in enumerate([5, 5, 5, 19, 1, 8]):
        k_new, v_new = synth.append_rows(3, 50 + s, w.B, w.Hkv, n_new)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16))
        c.decode_step(U.to_dev(w.q, torch.bfloat16), 0.9, out)
        torch.cuda.synchronize()
        assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all() and (c.n_total.cpu().numpy() == lazy.n_total).all()
        ref = orc.decode_step(w.q, lazy.K, lazy.V, lazy.codes, lazy.f_scale, None, lazy.c_k, None, lazy.n_indexed,
                              lazy.n_total, ROT_DENSE, rot128[0], 0.9, U.SM_SCALE)
        U.assert_attention_close(out.cpu().numpy(), ref["out"], "bf16")
    c.close()


def test_decode_step_host_buffers(orc, rot128):
    """rbq_decode_step_host: pinned host q in, host out; same bits as the device-buffer call."""
    import torch
    w = U.workload(1, L=2051)
    c = U.make_cache(w, rot128[0])
    c.encode_keys(U.to_dev(w.seq_lens))
    q_host = torch.from_numpy(w.q).to(torch.bfloat16).pin_memory()
    out_host = torch.zeros(w.B, w.Hq, 128, dtype=torch.float32).pin_memory()
    c.decode_step_host(q_host, 0.9, out_host)
    torch.cuda.synchronize()
    # on a non-default stream the host step is captured once and replayed as a CUDA graph: same result every time (up to the
    # accumulation order of S7, whose chunks are handed out dynamically)
    side = torch.cuda.Stream()
    outs = []
    for _ in range(4):
        o2 = torch.zeros_like(out_host).pin_memory()
        c.decode_step_host(q_host, 0.9, out_host if _ else o2, stream=side)
        side.synchronize()
        outs.append((out_host if _ else o2).clone())
    for o2 in outs[1:]:
        U.assert_same_step_output(o2.numpy(), outs[0].numpy(), "graph replay differs from the direct host step")
    out = c.new_out()
    c.decode_step(q_host.cuda(), 0.9, out)
    torch.cuda.synchronize()
    U.assert_same_step_output(out.cpu().numpy(), out_host.numpy())
    # new query values in the SAME pinned buffer (what a decode loop does): the replayed graph must read them afresh
    from paper_2606_31519_b200 import synth
    q_new = torch.from_numpy(synth.query_pool(w, 2)[1]).to(torch.bfloat16)
    q_host.copy_(q_new)
    c.decode_step_host(q_host, 0.9, out_host, stream=side)
    side.synchronize()
    c.decode_step(q_new.cuda(), 0.9, out)
    torch.cuda.synchronize()
    U.assert_same_step_output(out.cpu().numpy(), out_host.numpy())
    assert np.abs(out_host.numpy() - outs[0].numpy()).max() > 1e-2
    q_host.copy_(torch.from_numpy(w.q).to(torch.bfloat16))
    c.decode_step_host(q_host, 0.9, out_host, stream=side)
    side.synchronize()
    U.assert_same_step_output(out_host.numpy(), outs[0].numpy())
    # pageable host buffers take the staged path (pinned ones receive the result straight from the S7 merge)
    q_page = torch.from_numpy(w.q).to(torch.bfloat16).clone()
    out_page = torch.zeros(w.B, w.Hq, 128, dtype=torch.float32)
    assert not q_page.is_pinned() and not out_page.is_pinned()
    for st in (None, side):
        out_page.zero_()
        c.decode_step_host(q_page, 0.9, out_page, stream=st)
        (side if st is not None else torch.cuda.current_stream()).synchronize()
        U.assert_same_step_output(out_page.numpy(), out_host.numpy())
    assert c.launch_count() > 0
    c.close()


def test_error_codes(rot128):
    """Argument checks return negative status codes with a message; nothing is enqueued."""
    import ctypes as C
    import torch
    from paper_2606_31519_b200 import binding as rb
    rot = torch.from_numpy(rot128[0]).cuda()
    lib = rb.load()

    def create(**kw):
        base = dict(batch=1, n_q_heads=4, n_kv_heads=1, head_dim=128, max_tokens=256, flush_tokens=0, kv_dtype=1, q_dtype=1,
                    out_dtype=0, sm_scale=0.0, rot_kind=0, rot=rot.data_ptr(), enc_mode=0)
        base.update(kw)
        cfg = rb.rbq_config(**base)
        h = C.c_void_p()
        return lib.rbq_create(C.byref(cfg), C.byref(h)), h

    assert create(head_dim=96)[0] == -2 and create(head_dim=512)[0] == -2          # RBQ_ERR_UNSUPPORTED (64 / 128 / 256 are built)
    assert create(head_dim=64, enc_mode=1)[0] == -2 and create(head_dim=256, enc_mode=1)[0] == -2   # RBQ_ENC_FAST: head_dim 128 only
    assert create(n_q_heads=8, n_kv_heads=1)[0] == -2                               # G = 8
    assert create(head_dim=100)[0] == -1 and create(n_q_heads=3, n_kv_heads=2)[0] == -1
    assert create(max_tokens=0)[0] == -1 and create(rot=None)[0] == -1
    rc, h = create()
    assert rc == 0
    n = rb.rbq_workspace_bytes(h)
    assert n > 0
    # no workspace yet
    q = torch.zeros(1, 4, 128, dtype=torch.bfloat16, device="cuda")
    idx = rb.rbq_index(None, None, None, rot.data_ptr(), None, rot.data_ptr(), rot.data_ptr())
    assert lib.rbq_query_quantize(h, q.data_ptr(), C.byref(idx), None, None, None) == -3      # RBQ_ERR_WORKSPACE
    assert b"workspace" in lib.rbq_last_error(h)
    small = torch.zeros(256, dtype=torch.uint8, device="cuda")
    assert lib.rbq_set_workspace(h, small.data_ptr(), 256) == -3
    ws = torch.zeros(n, dtype=torch.uint8, device="cuda")
    assert lib.rbq_set_workspace(h, ws.data_ptr(), n) == 0
    assert lib.rbq_estimate_scores(h, q.data_ptr(), C.byref(idx), None, None) == -1           # codes / scores null
    with pytest.raises(rb.RbqError):
        rb.rbq_topp_select(h, q, idx, 0.0, q, q)                                              # p must be > 0
    assert lib.rbq_destroy(h) == 0


@pytest.mark.parametrize("cfg", [2, 3])
def test_full_size_configs(orc, rot128, cfg):
    """BASELINE.json configs 2 and 3 at FULL size (131 072-token context; 16 ragged sequences of 16 K - 64 K tokens), in the
    launch configuration bench.py times: the whole chain against the oracle (codes bit-exact inside _chained's encode
    check below, logits 1e-5, Top-p sets by the exact rule on the GPU's logits, outputs within tolerance)."""
    import torch
    w = U.workload(cfg)
    o = _chained(orc, w, rot128[0], ROT_DENSE, w.p)
    # codes and factors at full size, bit for bit
    c = U.make_cache(w, rot128[0])
    c.encode_keys(U.to_dev(w.seq_lens))
    torch.cuda.synchronize()
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    for b in range(w.B):
        n = int(w.seq_lens[b])
        assert (codes[b, :, :n] == o["codes"][b, :, :n]).all()
        assert (fs[b, :, :n].view(np.uint32) == o["f_scale"][b, :, :n].view(np.uint32)).all()
    c.close()


def test_config4_decode_loop_side_stream(orc, rot128):
    """BASELINE config 4 shape at a reduced context: batch 4, W = 64, 130 decode steps, each appending one token per
    sequence, the batched encode of every full window running on a side stream while the following decode step runs on
    the main stream (no host synchronisation between steps except at the checked ones)."""
    import torch
    from paper_2606_31519_b200 import synth
    W, steps = 64, 130
    w = U.workload(4, L=6000, B=4, extra_cap=192)
    rot = rot128[0]
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, ROT_DENSE, rot, W)
    c = U.make_cache(w, rot, flush_tokens=W)
    c.encode_keys(U.to_dev(w.seq_lens))
    main, side = torch.cuda.current_stream(), torch.cuda.Stream()
    pool = synth.query_pool(w, 4)
    q_dev = [U.to_dev(pool[i], torch.bfloat16) for i in range(4)]
    out = c.new_out()
    sel_cnt = c.new_sel()[1]
    check = {0, W - 2, W - 1, W, W + 1, 2 * W - 1, 2 * W, steps - 1}
    for s in range(steps):
        k_new, v_new = synth.append_rows(4, s, w.B, w.Hkv, 1)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16), stream=main, side_stream=side)
        c.decode_step(q_dev[s % 4], w.p, out, None, sel_cnt)
        if s in check:
            torch.cuda.synchronize()
            assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all() and (c.n_total.cpu().numpy() == lazy.n_total).all()
            ref = orc.decode_step(pool[s % 4], lazy.K, lazy.V, lazy.codes, lazy.f_scale, None, lazy.c_k, None, lazy.n_indexed,
                                  lazy.n_total, ROT_DENSE, rot, w.p, U.SM_SCALE)
            U.assert_attention_close(out.cpu().numpy(), ref["out"], "bf16")
            assert np.abs(sel_cnt.cpu().numpy().astype(np.int64) - ref["sel_cnt"]).max() <= max(2, int(0.002 * ref["sel_cnt"].max()))
    torch.cuda.synchronize()
    codes = c.codes.cpu().numpy().view(np.uint32)
    for b in range(w.B):
        n = int(lazy.n_indexed[b]) + lazy.in_flight
        assert (codes[b, :, :n] == lazy.codes[b, :, :n]).all()
    c.close()
