#!/usr/bin/env python
"""Benchmark of the RaBitQCache decode hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config 2]

A "step" is one pass of the whole hot path (S3 query prep -> S4/S5 estimator over the whole indexed
context -> S6 Top-p -> S7 gather attention) for one decode token of one attention layer of the
Llama-3.1-8B-shaped workload of BASELINE.json config 2 (32 q heads / 8 KV heads, D = 128, 131072 bf16
tokens, p = 0.9), seeded synthetic data (paper_2606_31519_b200.synth).  Cold L2: the steps rotate over
R independent layer replicas (distinct device buffers) whose combined touched footprint exceeds L2,
as the other layers of a model would between two visits of one layer.

Prints ONE JSON line (rank 0).  `value` = microseconds per decode step per layer, device-timed with CUDA
events, max over ranks, inputs resident in HBM.  `e2e` = the same through rbq_decode_step_host with
pinned HOST q / out buffers (copies inside the timed region, one stream sync per step).
`roofline` = dominant kernel: algorithmic bytes / CUDA-event duration vs the measured HBM peak.
`cpu_baseline` = the CPU oracle, as it stands, on the same workload (reported baseline, not the target).
`--impl reference` times the oracle alone (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "us_per_decode_step_per_layer_128k_ctx"
UNIT = "us"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0           # BASELINE.json quotes fractions of ~8 TB/s


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peak():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            return float(json.loads(f.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(stage: str):
    """DRAM bytes per launch of a stage's kernel from the committed ncu --set full capture, or None."""
    f = ROOT / "profiles" / "ncu_traffic.csv"
    if not f.exists():
        return None
    for line in f.read_text().splitlines():
        parts = [x.strip() for x in line.split(",")]
        if len(parts) >= 3 and parts[0] == stage:
            try:
                return float(parts[2])
            except ValueError:
                return None
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, device_index: int, period_s: float = 0.002):
        self.period, self.samples, self.reasons, self.sm_max = period_s, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:          # pragma: no cover
            log(f"[bench] NVML unavailable ({e}); clocks not sampled")

    def _once(self):
        nv = self.nv
        self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        for bit, name in self.REASONS.items():
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                break
            time.sleep(self.period)

    def __enter__(self):
        if self.h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
            try:
                self._once()
            except Exception:
                pass

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def build_workload(cfg_id: int, L: int | None):
    from paper_2606_31519_b200 import synth
    t0 = time.time()
    w = synth.make_workload(cfg_id, L=L)
    log(f"[bench] workload config {cfg_id}: B={w.B} Hq={w.Hq} Hkv={w.Hkv} L={w.seq_lens.tolist()} {w.kv_dtype} "
        f"p={w.p} generated in {time.time() - t0:.1f}s")
    return w


def workload_name(w):
    return (f"BASELINE config {w.cfg}: B={w.B}, {w.Hq} q heads / {w.Hkv} KV heads, D={w.D}, context "
            f"{int(w.seq_lens.max())}, {w.kv_dtype} K/V, top-p={w.p}")


# ---- CPU oracle arm (cpu_baseline leg and --impl reference) ---------------------------------------------
class OracleStep:
    """The oracle's decode step on (a sample of) the workload: index built once (untimed), then
    O3 -> O4 -> O5 -> O6 -> O7 per step.  sample = the first `n_kv` KV heads (with their query heads);
    the time is scaled by Hkv / n_kv to the full step."""

    def __init__(self, w, n_kv=None):
        from oracle import rbq_oracle as orc
        self.orc, self.w = orc, w
        self.n_kv = w.Hkv if n_kv is None else n_kv
        G = w.Hq // w.Hkv
        self.K = np.ascontiguousarray(w.K[:, :self.n_kv])
        self.V = np.ascontiguousarray(w.V[:, :self.n_kv])
        self.q = np.ascontiguousarray(w.q[:, :self.n_kv * G])
        self.rot, _ = orc.rotation_from_gaussian(w.rot_gauss)
        t0 = time.time()
        self.c_k = orc.centroid(self.K, w.seq_lens)
        self.codes, self.f_scale, _ = orc.encode(self.K, np.zeros_like(w.seq_lens), w.seq_lens, orc.ROT_DENSE, self.rot,
                                                 self.c_k)
        self.encode_s = time.time() - t0
        self.scale = w.Hkv / self.n_kv
        self.cores = orc.max_threads()

    def step(self):
        w = self.w
        return self.orc.decode_step(self.q, self.K, self.V, self.codes, self.f_scale, None, self.c_k, None, w.seq_lens,
                                    w.seq_lens, self.orc.ROT_DENSE, self.rot, w.p, 1.0 / math.sqrt(w.D))

    def sample_name(self):
        w = self.w
        return (f"{self.n_kv} of {w.Hkv} KV heads ({self.n_kv * w.Hq // w.Hkv} of {w.Hq} query heads) of the same workload, "
                f"full context, one oracle decode step per timed step, time scaled x{self.scale:g} to the full step")


def time_oracle(w, budget_s=12.0, n_kv=None, steps=None):
    o = OracleStep(w, n_kv)
    o.step()                                             # warm caches / page in
    ts = []
    t_begin = time.time()
    while True:
        t0 = time.perf_counter()
        o.step()
        ts.append(time.perf_counter() - t0)
        if steps is not None:
            if len(ts) >= steps:
                break
        elif time.time() - t_begin >= budget_s and len(ts) >= 3:
            break
    return o, ts


def run_reference(args):
    """--impl reference: the CPU oracle as it stands on the box's host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = build_workload(args.config, args.ctx)
    # bounded sample: calibrate on one full step, then keep K steps within ~120 s
    o_full = OracleStep(w)
    o_full.step()
    t0 = time.perf_counter()
    o_full.step()
    t_full = time.perf_counter() - t0
    n_kv = w.Hkv
    while n_kv > 1 and t_full * (n_kv / w.Hkv) * (args.steps + args.warmup) > 120.0:
        n_kv //= 2
    o = o_full if n_kv == w.Hkv else OracleStep(w, n_kv)
    for _ in range(args.warmup):
        o.step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step()
    dt = time.perf_counter() - t0
    us = dt / args.steps * o.scale * 1e6
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(w), "note": "CPU oracle (oracle/rbq_ref.c), fp64 logits/softmax/attention"},
            "cpu_baseline": {"value": us, "unit": UNIT, "cores": o.cores, "kind": "oracle", "sample": o.sample_name()},
            "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# ---- B200 arm --------------------------------------------------------------------------------------------
def union_rows(sel_idx, sel_cnt, n_indexed, n_total, Hkv):
    """Sum over (b, KV head) of |union_h I_h U pending| and sum over q heads of |I_h U pending| (diagnostics
    for the attention roofline bytes; numpy on the host, outside every timed region)."""
    B, Hq, _ = sel_idx.shape
    G = Hq // Hkv
    uni = per_head = 0
    for b in range(B):
        pend = int(n_total[b] - n_indexed[b])
        for g in range(Hkv):
            parts = [sel_idx[b, g * G + j, :sel_cnt[b, g * G + j]] for j in range(G)]
            uni += np.unique(np.concatenate(parts)).size + pend
            per_head += sum(p.size for p in parts) + G * pend
    return uni, per_head


def run_b200(args):
    import torch
    from paper_2606_31519_b200 import binding as rb
    from paper_2606_31519_b200 import dist as rdist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the RaBitQCache path has no CPU fallback")
    rank, local_rank, world = rdist.init_process_group("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    w = build_workload(args.config, args.ctx)
    dt = torch.float32 if w.kv_dtype == "f32" else torch.bfloat16
    rot = rb.make_rotation(31519)                       # product-side Haar rotation (host init)
    R = args.replicas
    caches = []
    K_dev = torch.from_numpy(w.K).to(dt).to(dev)
    V_dev = torch.from_numpy(w.V).to(dt).to(dev)
    seq_dev = torch.from_numpy(w.seq_lens).to(dev)
    for r in range(R):
        c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, rot, kv_dtype=dt, q_dtype=dt, out_dtype=torch.float32,
                           flush_tokens=w.flush_tokens)
        c.K.copy_(K_dev)
        c.V.copy_(V_dev)
        c.encode_keys(seq_dev)
        caches.append(c)
    del K_dev, V_dev
    torch.cuda.synchronize()
    q_dev = torch.from_numpy(w.q).to(dt).to(dev)
    outs = [c.new_out() for c in caches]
    sels = [c.new_sel() for c in caches]
    stream = torch.cuda.current_stream()

    def step(i):
        r = i % R
        caches[r].decode_step(q_dev, w.p, outs[r], None, sels[r][1])     # selection stays a bitmap in the workspace

    # ---- device-timed region: W warm-ups, then exactly K steps ---------------------------------------------
    for i in range(args.warmup):
        step(i)
    launches0 = sum(c.launch_count() for c in caches)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    rdist.barrier()
    with ClockSampler(local_rank) as clk:
        torch.cuda.synchronize()
        e0.record(stream)
        for i in range(args.steps):
            step(args.warmup + i)
        e1.record(stream)
        torch.cuda.synchronize()
    rdist.barrier()
    ms_total = e0.elapsed_time(e1)
    gpu_launches = sum(c.launch_count() for c in caches) - launches0
    # per-stage breakdown: a second, separate pass with the library's stage events between the kernels (the events
    # serialise the launches, so the stage times add up to a little more than the step timed above)
    for c in caches:
        c.profile_enable(True)
    for i in range(min(args.steps, 256)):
        step(args.warmup + i)
    torch.cuda.synchronize()
    stage_ms = {k: 0.0 for k in rb.STAGE_NAMES}
    n_prof = 0
    for c in caches:
        ms, n = c.profile_read()
        n_prof += n
        for k in ms:
            stage_ms[k] += ms[k]
        c.profile_enable(False)
    ms_total = rdist.max_over_ranks(ms_total, dev)
    us_step = ms_total * 1e3 / args.steps

    # ---- per-step distribution (diagnostic): K more steps, each between its own pair of events ------------
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(min(args.steps, 256))]
    for i, (a, b) in enumerate(evs):
        a.record(stream)
        step(i)
        b.record(stream)
    torch.cuda.synchronize()
    per_step = np.array([a.elapsed_time(b) * 1e3 for a, b in evs])

    # ---- end to end through the public host-buffer call ---------------------------------------------------
    q_host = torch.from_numpy(w.q).to(dt).pin_memory()
    out_host = torch.zeros(w.B, w.Hq, w.D, dtype=torch.float32).pin_memory()
    # on a non-default stream: the library replays the copies and the launches of a host step as one CUDA graph there
    e2e_stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    for i in range(max(args.warmup, 2 * R)):
        caches[i % R].decode_step_host(q_host, w.p, out_host, stream=e2e_stream)
        e2e_stream.synchronize()
    torch.cuda.synchronize()
    rdist.barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        caches[(args.warmup + i) % R].decode_step_host(q_host, w.p, out_host, stream=e2e_stream)
        e2e_stream.synchronize()                        # the model needs this layer's output before it goes on
    torch.cuda.synchronize()
    e2e_us = (time.perf_counter() - t0) * 1e6 / args.steps
    rdist.barrier()
    e2e_us = rdist.max_over_ranks(e2e_us, dev)

    # ---- roofline bookkeeping (host, untimed) -----------------------------------------------------------------
    caches[0].decode_step(q_dev, w.p, outs[0], sels[0][0], sels[0][1])   # untimed: index lists for the diagnostics below
    torch.cuda.synchronize()
    sel_idx = sels[0][0].cpu().numpy()
    sel_cnt = sels[0][1].cpu().numpy()
    n_idx = caches[0].n_indexed.cpu().numpy()
    n_tot = caches[0].n_total.cpu().numpy()
    uni, per_head = union_rows(sel_idx, sel_cnt, n_idx, n_tot, w.Hkv)
    esz = 2 if w.kv_dtype == "bf16" else 4
    alg = {
        "estimator": float(n_idx.sum()) * w.Hkv * (w.D // 8 + 4),          # 16 B code + 4 B factor per (token, KV head)
        "attn_gather": float(uni) * 2 * w.D * esz,                          # K row + V row per attended (token, KV head), union over the group
        "topp": float(n_idx.sum()) * w.Hq * 4,                              # one pass over the fp32 scores
    }
    peak, peak_src = measured_peak()
    stages = {}
    for k in rb.STAGE_NAMES:
        us = stage_ms[k] * 1e3 / max(1, n_prof)
        ent = {"us": us}
        if k in alg and us > 0:
            ent.update(bytes=alg[k], achieved_gbs=alg[k] / (us * 1e-6) / 1e9)
            ent.update(frac_measured=ent["achieved_gbs"] / peak, frac_8tbs=ent["achieved_gbs"] / NOMINAL_HBM_GBS)
        stages[k] = ent
    dom = max(("estimator", "attn_gather", "topp"), key=lambda k: stages[k]["us"])
    roofline = {"bound": "hbm", "kernel": dom, "achieved": stages[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": stages[dom]["achieved_gbs"] / peak, "traffic": ncu_traffic(dom), "peak_source": peak_src,
                "algorithmic_bytes": alg[dom], "us_per_launch": stages[dom]["us"], "stages": stages,
                "attended_rows_union": uni, "attended_rows_per_head_sum": per_head,
                "attn_per_head_bytes_gbs": per_head * 2 * w.D * esz / (stages["attn_gather"]["us"] * 1e-6) / 1e9
                if stages["attn_gather"]["us"] > 0 else None}

    line = None
    if rank == 0:
        clocks = clk.summary()
        budgets = sel_cnt.reshape(-1)
        line = {"metric": METRIC, "value": us_step / world, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16" if w.kv_dtype == "bf16" else "f32", "data": "synthetic",
                "config": {"workload": workload_name(w), "l2": f"cold: steps rotate over {R} layer replicas in distinct buffers "
                           f"({R * (2 * w.K.size * esz + alg['estimator']) / 2**30:.1f} GiB resident, L2 is 126 MB)",
                           "parallelism": f"{world} independent layer replica set(s), no data-path collective",
                           "budget_tokens": {"min": int(budgets.min()), "mean": float(budgets.mean()), "max": int(budgets.max())},
                           "value_note": "us per decode step per layer = max-over-ranks step time / n_gpus"},
                "clocks": clocks, "gpu_launches": int(gpu_launches),
                "step_us": {"p10": float(np.percentile(per_step, 10)), "median": float(np.median(per_step)),
                            "p90": float(np.percentile(per_step, 90))},
                "e2e": {"value": e2e_us / world, "unit": UNIT, "h2d_bytes_per_step": int(q_host.numel() * q_host.element_size()),
                        "d2h_bytes_per_step": int(out_host.numel() * out_host.element_size())},
                "roofline": roofline}
        if world == 1 and not args.no_cpu_baseline:
            o, ts = time_oracle(w, budget_s=args.cpu_seconds)
            line["cpu_baseline"] = {"value": float(np.median(ts)) * 1e6 * o.scale, "unit": UNIT, "cores": o.cores, "kind": "oracle",
                                    "sample": f"{len(ts)} full oracle decode steps of the same workload (median), index build "
                                              f"untimed ({o.encode_s:.1f}s)"}
        print(json.dumps(line), flush=True)
    for c in caches:
        c.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (2 = the 128K headline)")
    ap.add_argument("--ctx", type=int, default=None, help="override the context length (debug)")
    ap.add_argument("--replicas", type=int, default=8, help="layer replicas rotated over for cold-L2 timing")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
