"""Helpers shared by the `-m gpu` parity tests: upload a seeded workload into a RaBitQCache (CUDA path,
through the C ABI), run the CPU oracle on the same arrays, and the comparison rules of the
north_star (bit-exact integers / codes / factors, 1e-5 logits, Top-p sets identical up to boundary
tokens, 1e-2 / 2e-2 attention outputs for bf16 inputs).

Nothing here computes an expected value: expected values come from `oracle/` only.
"""
from __future__ import annotations

import functools
import math

import numpy as np

from paper_2606_31519_b200 import synth

D = 128
SM_SCALE = 1.0 / math.sqrt(D)


def sm_scale(w):
    return 1.0 / math.sqrt(w.D)


def torch_dtype(w):
    import torch
    return torch.float32 if w.kv_dtype == "f32" else torch.bfloat16


def to_dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)           # exact: bf16 workloads hold bf16-representable float32 values
    return t.cuda()


def make_cache(w, rot, *, rot_kind=0, with_cq=False, flush_tokens=0, out_dtype=None, upload_kv=True, **kw):
    """RaBitQCache for workload `w` with K/V (and c_q) uploaded; nothing encoded yet."""
    import torch
    from paper_2606_31519_b200 import binding as rb
    dt = torch_dtype(w)
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)),
                       flush_tokens=flush_tokens, kv_dtype=dt, q_dtype=dt, out_dtype=out_dtype or torch.float32,
                       rot_kind=rot_kind, with_cq=with_cq, head_dim=w.D, **kw)
    if upload_kv:
        c.K.copy_(to_dev(w.K, dt))
        c.V.copy_(to_dev(w.V, dt))
    if with_cq:
        c.c_q.copy_(to_dev(w.c_q))
    return c


def load_index(c, o):
    """Upload an oracle-made index (stage isolation: downstream GPU stages read the oracle's arrays)."""
    c.codes.copy_(to_dev(o["codes"].view(np.int32)))
    c.f_scale.copy_(to_dev(o["f_scale"]))
    c.c_k.copy_(to_dev(o["c_k"]))
    if o.get("f_bias") is not None and c.f_bias is not None:
        c.f_bias.copy_(to_dev(o["f_bias"]))
    c.n_indexed.copy_(to_dev(o["n_indexed"]))
    c.n_total.copy_(to_dev(o["n_total"]))


def oracle_index(orc, w, rot, rot_kind=0, with_cq=False, factor_f16=False):
    """O2: centroid + Alg.1 over tokens [0, seq_lens) with the oracle (factor_f16: O2c, factors rounded to binary16)."""
    c_k = orc.centroid(w.K, w.seq_lens)
    codes, f_scale, f_bias = orc.encode(w.K, np.zeros_like(w.seq_lens), w.seq_lens, rot_kind, rot, c_k,
                                        w.c_q if with_cq else None)
    if factor_f16:
        f_scale = orc.round_factors_f16(f_scale)
    return dict(c_k=c_k, codes=codes, f_scale=f_scale, f_bias=f_bias, n_indexed=w.seq_lens.copy(),
                n_total=w.seq_lens.copy())


def oracle_full(orc, w, rot, rot_kind=0, with_cq=False, p=None, factor_f16=False):
    o = oracle_index(orc, w, rot, rot_kind, with_cq, factor_f16)
    scores, qp, dot, pop = orc.estimate_scores(w.q, o["codes"], o["f_scale"], o["f_bias"], o["c_k"],
                                               w.c_q if with_cq else None, o["n_indexed"], rot_kind, rot, sm_scale(w))
    o.update(scores=scores, qp=qp, dot=dot, pop=pop)
    p = w.p if p is None else p
    n_rows = np.repeat(o["n_indexed"], w.Hq)
    sel_idx, sel_cnt = orc.topp(scores.reshape(w.B * w.Hq, w.Lcap), n_rows, p)
    o.update(sel_idx=sel_idx.reshape(w.B, w.Hq, w.Lcap), sel_cnt=sel_cnt.reshape(w.B, w.Hq), p=p)
    out, lse = orc.attention(w.q, w.K, w.V, o["sel_idx"], o["sel_cnt"], o["n_indexed"], o["n_total"], sm_scale(w))
    o.update(out=out, lse=lse)
    return o


@functools.lru_cache(maxsize=None)
def workload(cfg, L=None, B=None, variant="C", with_cq=False, extra_cap=0, n_heavy=None, D=128, Hq=None, Hkv=None):
    return synth.make_workload(cfg, L=L, B=B, variant=variant, with_cq=with_cq, extra_cap=extra_cap, n_heavy=n_heavy, D=D,
                               Hq=Hq, Hkv=Hkv)


@functools.lru_cache(maxsize=None)
def rotation(orc_mod, D, kind=0):
    """Rotation input of the recipe for head_dim D: dense QR matrix (kind 0, by the oracle) or WH sign vector (kind 1)."""
    if kind == 1:
        return synth.wh_sign_vector(D)
    return orc_mod.rotation_from_gaussian(synth.rotation_gaussian(D))[0]


# ---- comparison rules -------------------------------------------------------------------------------
def assert_logits_close(got, want, n_indexed, Hq):
    """|diff| <= 1e-5 * max(|oracle|, RMS of the row)   (north_star: 1e-5 relative in fp32)."""
    B = got.shape[0]
    for b in range(B):
        n = int(n_indexed[b])
        if n == 0:
            continue
        g = got[b, :, :n].astype(np.float64)
        o = want[b, :, :n].astype(np.float64)
        rms = np.sqrt((o ** 2).mean(axis=1, keepdims=True))
        tol = 1e-5 * np.maximum(np.abs(o), rms)
        bad = np.abs(g - o) > tol
        assert not bad.any(), f"seq {b}: {bad.sum()} logits off; worst {np.abs(g - o).max():.3e} (tol {tol.min():.3e})"


def softmax64(s):
    s = s.astype(np.float64)
    w = np.exp(s - s.max())
    return w / w.sum()


def assert_topp_row(scores_row, sel_gpu, sel_orc, p, slack=1e-6):
    """Identical sets, except tokens whose probability is within `slack` of the boundary probability or
    when the cumulative mass at the boundary is within `slack` of p; then the Top-p properties must hold
    with that slack."""
    sg, so = set(int(x) for x in sel_gpu), set(int(x) for x in sel_orc)
    assert len(sg) == len(sel_gpu), "duplicate indices in the GPU selection"
    if sg == so:
        return 0
    pr = softmax64(scores_row)
    diff = sorted(sg ^ so)
    pb = min(pr[list(so)]) if so else 0.0               # boundary probability of the oracle set
    mass_o = pr[list(so)].sum() if so else 0.0
    near_p = abs(mass_o - p) <= slack or abs(mass_o - pb - p) <= slack
    for t in diff:
        assert abs(pr[t] - pb) <= slack or near_p, f"token {t}: prob {pr[t]:.3e} vs boundary {pb:.3e}, mass {mass_o:.9f}"
    mask = np.zeros(len(scores_row), bool)
    mask[list(sg)] = True
    if not mask.all() and mask.any():
        assert pr[mask].min() >= pr[~mask].max() - slack
        m = pr[mask].sum()
        assert m >= p - slack and m - pr[mask].min() < p + slack
    return len(diff)


def assert_attention_close(got, want, kv_dtype):
    got = got.astype(np.float64)
    want = want.astype(np.float64)
    if kv_dtype == "f32":
        rtol, atol = 1e-4, 1e-4
    else:
        rtol, atol = 1e-2, 2e-2
    err = np.abs(got - want) - (rtol * np.abs(want) + atol)
    assert (err <= 0).all(), f"attention output off by up to {np.abs(got - want).max():.3e}"


def assert_same_step_output(a, b, msg=""):
    """Two runs of S7 on the same inputs: the bf16 tensor-pipe gather hands a KV group's chunks to its warps dynamically, so
    the fp32 accumulation ORDER (not the attended set) differs from run to run -- equal up to that rounding: 5e-5 of the
    output scale in fp32 (bf16 outputs: one bf16 ulp).  The deterministic paths (fp32, head_dim 256, RBQ_GATHER_PLAN=1)
    pass the same bound trivially."""
    a = np.asarray(a, dtype=np.float32) if a.dtype != np.float32 else a
    b = np.asarray(b, dtype=np.float32) if b.dtype != np.float32 else b
    scale = max(1.0, float(np.abs(b).max()))
    assert np.abs(a - b).max() <= 5e-5 * scale, msg or "outputs of two runs differ beyond accumulation order"
