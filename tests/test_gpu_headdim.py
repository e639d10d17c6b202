"""Head dims 64 and 256 (Table 5 has a D = 64 row, L534 "D generally >= 128"): every stage
of the path against the oracle at the same tolerances as D = 128 -- codes / factors / INT4 query codes / integer dots
bit-exact, logits 1e-5, Top-p by the exact rule on the GPU's logits, attention 1e-2 / 2e-2 (bf16) and 1e-4 (fp32),
lazy flush.  D = 64 runs the tensor-pipe gather, D = 256 the FP32-pipe attention kernel.
"""
import numpy as np
import pytest

from tests import gpu_util as U
from tests.test_gpu_chained import _chained

pytestmark = pytest.mark.gpu

ROT_DENSE, ROT_WH = 0, 1


def _unpack(codes):
    return ((codes[..., None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(codes.shape[:-1] + (-1,))


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("cfg,kw", [(0, dict(L=1111)), (1, dict(L=3001)), (3, dict(L=1500, B=3))])
@pytest.mark.parametrize("D", [64, 256])
def test_encode_keys_bit_exact_headdim(orc, D, cfg, kw, kind):
    import torch
    w = U.workload(cfg, D=D, **kw)
    rot = U.rotation(orc, D, kind)
    o = U.oracle_index(orc, w, rot, kind)
    c = U.make_cache(w, rot, rot_kind=kind)
    c.codes.fill_(-1)
    c.encode_keys(U.to_dev(w.seq_lens))
    torch.cuda.synchronize()
    assert (c.c_k.cpu().numpy().view(np.uint32) == o["c_k"].view(np.uint32)).all(), "centroid differs"
    codes = c.codes.cpu().numpy().view(np.uint32)
    fs = c.f_scale.cpu().numpy()
    assert codes.shape[-1] == D // 32
    for b in range(w.B):
        n = int(w.seq_lens[b])
        assert (codes[b, :, :n] == o["codes"][b, :, :n]).all(), f"codes differ (seq {b})"
        assert (fs[b, :, :n].view(np.uint32) == o["f_scale"][b, :, :n].view(np.uint32)).all(), "f_scale differs"
        assert (codes[b, :, n:] == 0xFFFFFFFF).all(), "encode wrote beyond seq_len"
    c.close()


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("D", [64, 256])
def test_query_and_integer_dot_headdim(orc, D, kind):
    """S3 + S4: INT4 query codes and constants bit-exact; integer dots exact, including single-bit codes that must read
    back the INT4 query itself (checks the bit <-> MMA-operand mapping of every dimension)."""
    import torch
    w = U.workload(1, L=1500, D=D, with_cq=True)
    rot = U.rotation(orc, D, kind)
    o = U.oracle_index(orc, w, rot, kind, with_cq=True)
    qp = orc.query_prep(w.q, w.Hkv, kind, rot, o["c_k"], w.c_q)
    W = D // 32
    rng = np.random.default_rng(D)
    codes = rng.integers(0, 2 ** 32, (w.B, w.Hkv, w.Lcap, W), dtype=np.uint64).astype(np.uint32)
    codes[:, :, 0] = 0
    codes[:, :, 1] = 0xFFFFFFFF
    for j in range(D):
        codes[:, :, 4 + j] = 0
        codes[:, :, 4 + j, j // 32] = np.uint32(1) << np.uint32(j % 32)
    o["codes"] = codes
    d_ref, p_ref = orc.int_dots(codes, qp["qu"], w.seq_lens)
    c = U.make_cache(w, rot, rot_kind=kind, with_cq=True, upload_kv=False)
    U.load_index(c, o)
    qu = torch.zeros(w.B, w.Hq, D, dtype=torch.uint8, device="cuda")
    par = torch.zeros(w.B, w.Hq, 6, dtype=torch.float32, device="cuda")
    q = U.to_dev(w.q, U.torch_dtype(w))
    c.query_quantize(q, qu, par)
    dot = torch.zeros(w.B, w.Hq, w.Lcap, dtype=torch.int32, device="cuda")
    pop = torch.zeros(w.B, w.Hkv, w.Lcap, dtype=torch.int32, device="cuda")
    c.int4_dot_binary(q, dot, pop)
    torch.cuda.synchronize()
    assert (qu.cpu().numpy() == qp["qu"]).all(), "INT4 query codes differ"
    par = par.cpu().numpy()
    for i, key in enumerate(["qn", "ql", "delta"]):
        assert (par[..., i].view(np.uint32) == qp[key].view(np.uint32)).all(), key
    assert (par[..., 3] == qp["sumq"]).all()
    assert (par[..., 4].view(np.uint32) == qp["q_ck"].view(np.uint32)).all()
    assert (par[..., 5].view(np.uint32) == qp["cq_ck"].view(np.uint32)).all()
    L = int(w.seq_lens[0])
    assert (dot.cpu().numpy()[..., :L] == d_ref[..., :L]).all()
    assert (pop.cpu().numpy()[..., :L] == p_ref[..., :L]).all()
    assert (dot.cpu().numpy()[0, :, 4:4 + D] == qp["qu"][0]).all()
    c.close()


@pytest.mark.parametrize("kind", [ROT_DENSE, ROT_WH])
@pytest.mark.parametrize("cfg,kw,p", [(0, dict(L=2049), 0.9), (1, dict(L=5003), 0.9), (2, dict(L=6150, n_heavy=32), 0.8),
                                      (3, dict(L=3001, B=3), 0.95)])
@pytest.mark.parametrize("D", [64, 256])
def test_decode_step_chained_headdim(orc, D, cfg, kw, p, kind):
    _chained(orc, U.workload(cfg, D=D, **kw), U.rotation(orc, D, kind), kind, p)


@pytest.mark.parametrize("D", [64, 256])
def test_decode_step_chained_with_cq_headdim(orc, D):
    _chained(orc, U.workload(1, L=2500, D=D, with_cq=True), U.rotation(orc, D), ROT_DENSE, 0.9, with_cq=True)


@pytest.mark.parametrize("D", [64, 256])
def test_p1_is_dense_attention_headdim(orc, D):
    import torch
    w = U.workload(1, L=2051, D=D)
    c = U.make_cache(w, U.rotation(orc, D))
    c.encode_keys(U.to_dev(w.seq_lens))
    q = U.to_dev(w.q, torch.bfloat16)
    out = c.new_out()
    c.decode_step(q, 1.0, out)
    torch.cuda.synchronize()
    G = w.Hq // w.Hkv
    n = int(w.seq_lens[0])
    kk = c.K[0, :, :n].float().repeat_interleave(G, dim=0)
    vv = c.V[0, :, :n].float().repeat_interleave(G, dim=0)
    sd = torch.nn.functional.scaled_dot_product_attention(q[0].float()[:, None, :], kk, vv)[:, 0]
    U.assert_attention_close(out[0].cpu().numpy(), sd.cpu().numpy(), "bf16")
    c.close()


@pytest.mark.parametrize("D", [64, 256])
def test_append_flush_headdim(orc, D):
    """Lazy updates (L215) at D = 64 / 256: W = 8, 1 token per step, side stream; counts, codes of flushed rows, outputs."""
    import torch
    from paper_2606_31519_b200 import synth
    W, steps = 8, 19
    w = U.workload(3, L=900, B=3, extra_cap=64, D=D)
    rot = U.rotation(orc, D)
    lazy = orc.LazyIndex(w.K, w.V, w.seq_lens, ROT_DENSE, rot, W)
    c = U.make_cache(w, rot, flush_tokens=W)
    c.encode_keys(U.to_dev(w.seq_lens))
    side = torch.cuda.Stream()
    out = c.new_out()
    sel_cnt = c.new_sel()[1]
    for s in range(steps):
        k_new, v_new = synth.append_rows(3, s, w.B, w.Hkv, 1, D=D)
        lazy.append(k_new, v_new)
        c.append_tokens(U.to_dev(k_new, torch.bfloat16), U.to_dev(v_new, torch.bfloat16), side_stream=side)
        c.decode_step(U.to_dev(w.q, torch.bfloat16), 0.9, out, None, sel_cnt)
        torch.cuda.synchronize()
        assert (c.n_indexed.cpu().numpy() == lazy.n_indexed).all() and (c.n_total.cpu().numpy() == lazy.n_total).all()
        if s in (0, W - 1, W, 2 * W, steps - 1):
            ref = orc.decode_step(w.q, lazy.K, lazy.V, lazy.codes, lazy.f_scale, None, lazy.c_k, None, lazy.n_indexed,
                                  lazy.n_total, ROT_DENSE, rot, 0.9, U.sm_scale(w))
            U.assert_attention_close(out.cpu().numpy(), ref["out"], "bf16")
            assert np.abs(sel_cnt.cpu().numpy().astype(np.int64) - ref["sel_cnt"]).max() <= 2
    codes = c.codes.cpu().numpy().view(np.uint32)
    for b in range(w.B):
        n = int(lazy.n_indexed[b]) + lazy.in_flight
        assert (codes[b, :, :n] == lazy.codes[b, :, :n]).all()
    c.close()
