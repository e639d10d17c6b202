"""Micro-benchmarks of the paths bench.py does not time (the setup path S1 and the alternative Top-p selector).

    python -m paper_2606_31519_b200.microbench encode [--reps 5]     # rbq_encode_keys, 8 KV heads x 131 072 bf16 keys
    python -m paper_2606_31519_b200.microbench alg3   [--reps 20]    # rbq_topp_select vs rbq_topp_select_alg3, config 2

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
                                ("Walsh-Hadamard RBQ_ENC_EXACT", wh, rb.RBQ_ROT_WH, rb.RBQ_ENC_EXACT)):
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


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("what", choices=["encode", "alg3"])
    ap.add_argument("--reps", type=int, default=0)
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("microbench needs a GPU (there is no CPU fallback)")
    if a.what == "encode":
        encode(a.reps or 5)
    else:
        alg3(a.reps or 20)


if __name__ == "__main__":
    main()
