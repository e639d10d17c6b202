"""Micro-benchmarks of the paths bench.py does not time (the setup path S1 and the alternative Top-p selector).

    python -m paper_2606_31519_b200.microbench encode [--reps 5]     # rbq_encode_keys, 8 KV heads x 131 072 bf16 keys
    python -m paper_2606_31519_b200.microbench alg3   [--reps 20]    # rbq_topp_select vs rbq_topp_select_alg3, config 2
    python -m paper_2606_31519_b200.microbench prefill [--reps N]    # index build on a side stream under a dense prefill

Inputs are seeded and synthetic (synth.py); timing is by CUDA events on the current stream after warm-up.  These are
the commands the ncu captures of profiles/r01e_ncu_full.md profile.
"""
import argparse

import numpy as np
import torch

from . import binding as rb
from . import synth


def _time_us(fn, reps, warm=3):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e3 / reps


def encode(reps):
    B, Hq, Hkv, L = 1, 32, 8, 131072
    rot = rb.make_rotation(31519)
    wh = torch.from_numpy(synth.wh_sign_vector(128).astype(np.float32))
    g = torch.Generator(device="cuda").manual_seed(31519)
    K = torch.randn(B, Hkv, L, 128, device="cuda", generator=g).to(torch.bfloat16)
    sl = torch.full((B,), L, dtype=torch.int32, device="cuda")
    units = B * Hkv * L
    for name, r, kind, mode in (("dense RBQ_ENC_EXACT", rot, rb.RBQ_ROT_DENSE, rb.RBQ_ENC_EXACT),
                                ("dense RBQ_ENC_FAST", rot, rb.RBQ_ROT_DENSE, rb.RBQ_ENC_FAST),
                                ("Walsh-Hadamard RBQ_ENC_EXACT", wh, rb.RBQ_ROT_WH, rb.RBQ_ENC_EXACT),
                                ("Walsh-Hadamard RBQ_ENC_FAST", wh, rb.RBQ_ROT_WH, rb.RBQ_ENC_FAST)):
        c = rb.RaBitQCache(B, Hq, Hkv, L, r, rot_kind=kind, enc_mode=mode)
        c.K.copy_(K)
        full = _time_us(lambda: c.encode_keys(sl), reps, warm=2)
        only = _time_us(lambda: c.encode_keys(sl, flags=rb.RBQ_CK_GIVEN), reps, warm=2)
        print(f"{name}: rbq_encode_keys {full:.0f} us (centroid + encode), encode only (RBQ_CK_GIVEN) {only:.0f} us; "
              f"{units / full:.0f} Munits/s, {units * 276 / full / 1e6:.2f} TB/s of 276 B/unit", flush=True)
        c.close()


def alg3(reps):
    w = synth.make_workload(2)
    dt = torch.bfloat16
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, rb.make_rotation(31519), kv_dtype=dt, q_dtype=dt, out_dtype=torch.float32)
    c.K.copy_(torch.from_numpy(w.K).to(dt).cuda())
    c.V.copy_(torch.from_numpy(w.V).to(dt).cuda())
    c.encode_keys(torch.from_numpy(w.seq_lens).cuda())
    q = torch.from_numpy(w.q).to(dt).cuda()
    scores = torch.empty((w.B, w.Hq, w.Lcap), dtype=torch.float32, device="cuda")
    c.estimate_scores(q, scores)
    idx_a, cnt_a = c.new_sel()
    idx_b, cnt_b = c.new_sel()
    iters = torch.zeros((w.B, w.Hq), dtype=torch.int32, device="cuda")
    for p in (0.8, 0.9, 0.95):
        ta = _time_us(lambda: c.topp_select(scores, p, idx_a, cnt_a), reps)
        tb = _time_us(lambda: c.topp_select_alg3(scores, p, idx_b, cnt_b, iters), reps)
        torch.cuda.synchronize()
        print(f"p={p}: rbq_topp_select {ta:.1f} us; rbq_topp_select_alg3 {tb:.1f} us; Alg.3 iterations min/mean/max "
              f"{int(iters.min())}/{float(iters.float().mean()):.1f}/{int(iters.max())}; selected {int(cnt_a.sum())} / "
              f"{int(cnt_b.sum())}", flush=True)
    c.close()


def prefill(reps):
    """Asynchronous pipelined prefill ("<10 % TTFT overhead"): the O(L^2) causal
    prefill attention of one layer (a library call, torch SDPA, standing in for the model) on a high-priority stream,
    rbq_encode_keys (centroid + Alg.1) of the same layer's keys on a second, lower-priority stream."""
    import torch.nn.functional as F
    Hq, Hkv = 32, 8
    rot = rb.make_rotation(31519)
    for L in (32768, 131072):
        n_rep = reps or (20 if L <= 32768 else 3)
        for mode, mname in ((rb.RBQ_ENC_EXACT, "RBQ_ENC_EXACT"), (rb.RBQ_ENC_FAST, "RBQ_ENC_FAST")):
            c = rb.RaBitQCache(1, Hq, Hkv, L, rot, enc_mode=mode)
            g = torch.Generator(device="cuda").manual_seed(L)
            c.K.copy_(torch.randn(1, Hkv, L, 128, device="cuda", generator=g).to(torch.bfloat16))
            c.V.copy_(torch.randn(1, Hkv, L, 128, device="cuda", generator=g).to(torch.bfloat16))
            q = torch.randn(1, Hq, L, 128, device="cuda", generator=g).to(torch.bfloat16)
            k, v = c.K.contiguous(), c.V.contiguous()
            sl = torch.full((1,), L, dtype=torch.int32, device="cuda")
            main, side = torch.cuda.Stream(priority=-1), torch.cuda.Stream(priority=0)

            def attn():
                with torch.cuda.stream(main):
                    return F.scaled_dot_product_attention(q, k, v, is_causal=True, enable_gqa=True)

            def run(with_attn, with_enc):
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(main)
                side.wait_event(e0)
                for _ in range(n_rep):
                    if with_attn:
                        attn()
                    if with_enc:
                        c.encode_keys(sl, stream=side)
                done = torch.cuda.Event()
                done.record(side)
                main.wait_event(done)
                e1.record(main)
                torch.cuda.synchronize()
                return e0.elapsed_time(e1) * 1e3 / n_rep

            run(True, True)
            ta, te, tb = run(True, False), run(False, True), run(True, True)
            print(f"L={L} {mname}: prefill attention {ta:.0f} us; index build alone {te:.0f} us; both (index build on the "
                  f"low-priority stream) {tb:.0f} us: overhead {100 * (tb - ta) / ta:+.2f} % of the attention "
                  f"(serial would be {100 * te / ta:+.2f} %)", flush=True)
            c.close()
            del q, k, v


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("what", choices=["encode", "alg3", "prefill"])
    ap.add_argument("--reps", type=int, default=0)
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("microbench needs a GPU (there is no CPU fallback)")
    if a.what == "encode":
        encode(a.reps or 5)
    elif a.what == "alg3":
        alg3(a.reps or 20)
    else:
        prefill(a.reps)


if __name__ == "__main__":
    main()
