"""rbq_topp_select_static: the Top-p selection (S6, Alg.2 line 12) for callers that cannot allocate device memory
or hand over a workspace -- its scratch is a static 2 MiB device array inside the library (include/rbq.h).

Collected last on purpose (the suite runs with `pytest -x`).  The new entry point must return exactly what the existing
path (`rbq_topp_select`, workspace-backed) returns -- index work: bit for bit -- on two calls in a row that share the
static array (the second with shorter rows, other scores and another p, so that stale contents of the first would show), from
a context that never received a workspace; and it must reject sizes beyond the array with a clear error.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _raw_ctx(rb, torch, B, Hq, Hkv, L, rot):
    """A context WITHOUT workspace (rbq_set_workspace never called) and the minimal index the selection needs."""
    cfg = rb.rbq_config(B, Hq, Hkv, 128, L, 0, rb._dt(torch.bfloat16), rb._dt(torch.bfloat16), rb._dt(torch.float32), 0.0,
                        rb.RBQ_ROT_DENSE, rot.data_ptr(), rb.RBQ_ENC_EXACT, rb.RBQ_F32)
    ctx = rb.rbq_create(cfg)
    c_k = torch.zeros(B, Hkv, 128, dtype=torch.float32, device="cuda")
    n_indexed = torch.zeros(B, dtype=torch.int32, device="cuda")
    n_total = torch.zeros(B, dtype=torch.int32, device="cuda")
    idx = rb.rbq_index(None, None, None, c_k.data_ptr(), None, n_indexed.data_ptr(), n_total.data_ptr())
    return ctx, idx, (c_k, n_indexed, n_total, cfg)


@pytest.mark.parametrize("B,Hq,Hkv,L", [(1, 32, 8, 40000), (3, 8, 2, 9000), (20, 8, 2, 2100)])
def test_static_scratch_topp_matches_workspace_path(rot128, B, Hq, Hkv, L):
    import torch
    from paper_2606_31519_b200 import binding as rb
    rot = torch.from_numpy(rot128[0]).cuda().contiguous()
    ref = rb.RaBitQCache(B, Hq, Hkv, L, rot)                       # existing path: context + workspace
    ctx, idx, keep = _raw_ctx(rb, torch, B, Hq, Hkv, L, rot)       # new path: no workspace at all
    n_indexed, n_total = keep[1], keep[2]
    g = torch.Generator(device="cuda")
    g.manual_seed(1000 + B)
    rng = np.random.default_rng(7 + B)
    calls = [(0.9, np.full(B, L, np.int32)),
             (0.6, rng.integers(max(1, L // 5), max(2, L // 2), B).astype(np.int32))]
    for k, (p, lens) in enumerate(calls):
        scores = torch.randn(B, Hq, L, device="cuda", generator=g) * (1.0 + 4.0 * torch.rand(B, Hq, 1, device="cuda", generator=g))
        scores[0, 0] = torch.round(scores[0, 0] * 2) / 2            # heavy ties: the cut is decided by the index order
        for t in (ref.n_indexed, ref.n_total, n_indexed, n_total):
            t.copy_(torch.from_numpy(lens))
        want_idx, want_cnt = ref.new_sel()
        got_idx, got_cnt = ref.new_sel()
        got_idx.fill_(-7)
        ref.topp_select(scores, p, want_idx, want_cnt)
        rb.rbq_topp_select_static(ctx, scores, idx, p, got_idx, got_cnt)
        torch.cuda.synchronize()
        wc, gc = want_cnt.cpu().numpy(), got_cnt.cpu().numpy()
        assert (wc == gc).all(), f"call {k}: budgets differ"
        assert (gc > 0).all() and (gc <= lens[:, None]).all()
        wi, gi = want_idx.cpu().numpy(), got_idx.cpu().numpy()
        for b in range(B):
            for h in range(Hq):
                n = int(gc[b, h])
                assert (wi[b, h, :n] == gi[b, h, :n]).all(), f"call {k}: selected set of row ({b}, {h}) differs"
    rb.rbq_destroy(ctx)
    ref.close()


def test_static_scratch_rejects_sizes_beyond_the_array(rot128):
    import torch
    from paper_2606_31519_b200 import binding as rb
    rot = torch.from_numpy(rot128[0]).cuda().contiguous()
    B, Hq, Hkv, L = 16, 32, 8, 65536                                # config 3: 512 rows x 2 048 words = 4 MiB > 2 MiB
    ctx, idx, keep = _raw_ctx(rb, torch, B, Hq, Hkv, L, rot)
    scores = torch.zeros(16, dtype=torch.float32, device="cuda")   # never read: the size check comes first
    sel = torch.zeros(16, dtype=torch.int32, device="cuda")
    with pytest.raises(rb.RbqError) as e:
        rb.rbq_topp_select_static(ctx, scores, idx, 0.9, sel, sel)
    assert "static array" in str(e.value) and "status" in str(e.value)
    rb.rbq_destroy(ctx)
