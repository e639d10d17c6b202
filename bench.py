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


NCU_SUMMARY = "profiles/ncu_summary.csv"


def ncu_summary():
    """{stage: (kernel, dram bytes per launch, us per launch)} from the COMMITTED ncu summary (a static file written from
    the captures named in profiles/*.md: not measured in this run -- `traffic_source` in the JSON line says so)."""
    f = ROOT / NCU_SUMMARY
    out = {}
    if not f.exists():
        return out
    for line in f.read_text().splitlines():
        parts = [x.strip() for x in line.split(",")]
        if len(parts) >= 4 and not parts[0].startswith("#"):
            try:
                out[parts[0]] = (parts[1], float(parts[2]), float(parts[3]))
            except ValueError:
                pass
    return out


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

    # ---- set-up, untimed: every replica decodes twice (S7 sizes its work partition with the union sizes it counted in the
    #      previous step of the same cache: the first step after rbq_set_workspace runs without that history) ------------
    for i in range(2 * R):
        step(i)
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
    ncu = ncu_summary()
    for k in rb.STAGE_NAMES:
        us = stage_ms[k] * 1e3 / max(1, n_prof)
        ent = {"us": us}
        if k in ncu:
            ent["us_ncu"] = ncu[k][2]               # committed launch list: cold-cache, serialised (compare shares)
        if k in alg and us > 0:
            ent.update(bytes=alg[k], achieved_gbs=alg[k] / (us * 1e-6) / 1e9)
            ent.update(frac_measured=ent["achieved_gbs"] / peak, frac_8tbs=ent["achieved_gbs"] / NOMINAL_HBM_GBS)
        stages[k] = ent
    dom = max(("estimator", "attn_gather", "topp"), key=lambda k: stages[k]["us"])
    roofline = {"bound": "hbm", "kernel": dom, "achieved": stages[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": stages[dom]["achieved_gbs"] / peak, "traffic": ncu[dom][1] if dom in ncu else None,
                "traffic_source": f"static: {NCU_SUMMARY} (committed ncu --set full capture, not measured in this run)",
                "frac_at_ncu_duration": (alg[dom] / (ncu[dom][2] * 1e-6) / 1e9 / peak) if dom in ncu else None,
                "peak_source": peak_src,
                "kernel_note": ("attn_gather = the whole S7 stage in ONE kernel (attn_gather_bits_kernel: expands the selection "
                                "bitmaps, gathers, contracts, merges); until the middle of round 2 S7 was attn_plan + attn_gather "
                                "and this entry was the second of the two kernels only") if dom == "attn_gather" else None,
                "algorithmic_bytes": alg[dom], "us_per_launch": stages[dom]["us"], "stages": stages,
                "attended_rows_union": uni, "attended_rows_per_head_sum": per_head,
                "attn_per_head_bytes_gbs": per_head * 2 * w.D * esz / (stages["attn_gather"]["us"] * 1e-6) / 1e9
                if stages["attn_gather"]["us"] > 0 else None}

    # warm-L2 variant of the same step (labelled as such): one replica, back to back
    o_w = caches[0].new_out()
    warm_us = ev_time_us(lambda i: caches[0].decode_step(q_dev, w.p, o_w), min(args.steps, 200), 5)
    try:
        recall = leg_recall(w, caches[0], q_dev, sel_idx, sel_cnt) if rank == 0 else None
    except Exception as e:                          # a diagnostic: never takes the headline down
        recall = {"error": f"{type(e).__name__}: {e}"}
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
                           "value_note": "us per decode step per layer = max-over-ranks step time / n_gpus",
                           "setup_note": "every layer replica decodes twice, untimed, before the W warm-up steps (steady state of a "
                                         "decode loop: S7 partitions its work with the union sizes counted in the replica's previous step)"},
                "clocks": clocks, "gpu_launches": int(gpu_launches),
                "step_us": {"p10": float(np.percentile(per_step, 10)), "median": float(np.median(per_step)),
                            "p90": float(np.percentile(per_step, 90))},
                "e2e": {"value": e2e_us / world, "unit": UNIT, "h2d_bytes_per_step": int(q_host.numel() * q_host.element_size()),
                        "d2h_bytes_per_step": int(out_host.numel() * out_host.element_size())},
                "roofline": roofline,
                "warm_l2_us": warm_us,                       # same step, ONE replica back to back: codes and much of K/V stay in L2
                "attention_recall": recall}
        for c in caches[1:]:                                 # the legs need the memory
            c.close()
        caches = caches[:1]
        torch.cuda.empty_cache()
        if world == 1 and args.legs:
            line["configs"] = run_legs(args, rb, w, rot, peak)
        if world == 1 and not args.no_cpu_baseline:
            o, ts = time_oracle(w, budget_s=args.cpu_seconds)
            line["cpu_baseline"] = {"value": float(np.median(ts)) * 1e6 * o.scale, "unit": UNIT, "cores": o.cores, "kind": "oracle",
                                    "sample": f"{len(ts)} full oracle decode steps of the same workload (median), index build "
                                              f"untimed ({o.encode_s:.1f}s)"}
            if args.legs:
                line["cpu_baseline"]["per_stage"] = cpu_stage_baseline(w)
        print(json.dumps(line), flush=True)
    for c in caches:
        c.close()
    return 0


# ---- measurement legs beside the headline (configs 0, 1, 3, 4, Table 5 shapes, 8(f) rows) --------------
# Every leg returns a small dict that goes under "configs" in the one JSON line; a leg that fails reports {"error": ...}
# and never takes the headline down.  All timings: CUDA events on the launching stream, after warm-up.
L2_BYTES = 126 * 2 ** 20
PAPER_T5 = [  # PAPER.md L361-372 (Table 5), "Warp" / "Original" kernel latency in ms on an unnamed Hopper GPU
    ((1, 1024, 8, 128), 0.0127, 0.0382), ((1, 4096, 8, 128), 0.0130, 0.0386), ((1, 8192, 8, 128), 0.0129, 0.0385),
    ((1, 16384, 8, 128), 0.0136, 0.0388), ((4, 4096, 8, 128), 0.0130, 0.0387), ((8, 4096, 8, 128), 0.0216, 0.0741),
    ((1, 4096, 32, 128), 0.0501, 0.1585), ((1, 8192, 8, 64), 0.0093, 0.0212)]


def ev_time_us(fn, n, warm=5):
    """us per call of fn(i): n calls between two CUDA events on the current stream, after `warm` untimed calls."""
    import torch
    for i in range(warm):
        fn(i)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for i in range(n):
        fn(warm + i)
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) * 1e3 / n


def make_replicas(rb, w, rot, R, **kw):
    """R independent caches holding workload w, encoded; K/V uploaded once and copied device-to-device."""
    import torch
    dt = torch.float32 if w.kv_dtype == "f32" else torch.bfloat16
    dev = torch.device("cuda")
    K_dev, V_dev = torch.from_numpy(w.K).to(dt).to(dev), torch.from_numpy(w.V).to(dt).to(dev)
    seq_dev = torch.from_numpy(w.seq_lens).to(dev)
    caches = []
    for _ in range(R):
        c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, rot, head_dim=w.D, kv_dtype=dt, q_dtype=dt, out_dtype=torch.float32,
                           flush_tokens=w.flush_tokens, **kw)
        c.K.copy_(K_dev)
        c.V.copy_(V_dev)
        c.encode_keys(seq_dev)
        caches.append(c)
    torch.cuda.synchronize()
    return caches, dt


def step_profile(rb, caches, q_dev, p, steps, warm=5):
    """us per decode step (events) + per-stage us (library stage events, separate pass) rotating over the replicas."""
    import torch
    R = len(caches)
    outs = [c.new_out() for c in caches]
    us = ev_time_us(lambda i: caches[i % R].decode_step(q_dev, p, outs[i % R]), steps, max(warm, 2 * R))   # >= 2 steps per replica first
    for c in caches:
        c.profile_enable(True)
    for i in range(min(steps, 128)):
        caches[i % R].decode_step(q_dev, p, outs[i % R])
    torch.cuda.synchronize()
    st, n = {k: 0.0 for k in rb.STAGE_NAMES}, 0
    for c in caches:
        ms, k = c.profile_read()
        n += k
        for key in ms:
            st[key] += ms[key]
        c.profile_enable(False)
    return us, {k: v * 1e3 / max(1, n) for k, v in st.items()}


def leg_static_config(rb, cfg_id, ps, rot, steps, peak):
    """Configs 0 and 1: the decode step at every p the config names; estimator / gather achieved GB/s and fractions."""
    import torch
    w = build_workload(cfg_id, None)
    esz = 2 if w.kv_dtype == "bf16" else 4
    per_replica = 2 * w.K.size * esz
    R = int(min(32, max(2, math.ceil(4 * L2_BYTES / per_replica))))
    caches, dt = make_replicas(rb, w, rot, R)
    q_dev = torch.from_numpy(w.q).to(dt).cuda()
    out = {"workload": workload_name(w), "l2": f"cold: {R} replicas, {R * per_replica / 2**20:.0f} MiB of K/V", "per_p": {}}
    sel = caches[0].new_sel()
    o0 = caches[0].new_out()
    for p in ps:
        us, st = step_profile(rb, caches, q_dev, p, steps)
        caches[0].decode_step(q_dev, p, o0, sel[0], sel[1])
        torch.cuda.synchronize()
        uni, per_head = union_rows(sel[0].cpu().numpy(), sel[1].cpu().numpy(), caches[0].n_indexed.cpu().numpy(),
                                   caches[0].n_total.cpu().numpy(), w.Hkv)
        est_b = float(w.seq_lens.sum()) * w.Hkv * (w.D // 8 + 4)
        att_b = float(uni) * 2 * w.D * esz
        ent = {"us_per_step": us, "stages_us": st, "budget_mean_tokens": float(sel[1].float().mean().item()),
               "estimator": {"bytes": est_b, "gbs": est_b / st["estimator"] / 1e3, "frac_measured": est_b / st["estimator"] / 1e3 / peak},
               "attn_gather": {"bytes": att_b, "gbs": att_b / st["attn_gather"] / 1e3, "frac_measured": att_b / st["attn_gather"] / 1e3 / peak}}
        out["per_p"][str(p)] = ent
    for c in caches:
        c.close()
    return out


def leg_table5(rb, steps):
    """PAPER.md Table 5 (L361-372): Int4DotBinary on the paper's eight shapes (batch, tokens, heads, head_size), Hq = Hkv,
    random codes and queries; S4/S5 alone = (S3 + S4/S5) - S3, both measured; cold L2 over 16 replicas."""
    import torch
    rows = []
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    for (B, L, H, D), warp_ms, orig_ms in PAPER_T5:
        R = 16
        rot = rb.make_rotation(31519, D)
        caches = []
        for _ in range(R):
            c = rb.RaBitQCache(B, H, H, L, rot, head_dim=D)
            c.codes.copy_(torch.randint(-2 ** 31, 2 ** 31 - 1, c.codes.shape, dtype=torch.int32, device="cuda", generator=g))
            c.f_scale.copy_(torch.rand(c.f_scale.shape, device="cuda", generator=g) + 0.5)
            c.n_indexed.fill_(L)
            c.n_total.fill_(L)
            caches.append(c)
        q = torch.randn(B, H, D, device="cuda", generator=g).to(torch.bfloat16)
        sc = [c.new_scores() for c in caches]
        t_q = ev_time_us(lambda i: caches[i % R].query_quantize(q), steps)
        t_qe = ev_time_us(lambda i: caches[i % R].estimate_scores(q, sc[i % R]), steps)
        units = B * H * L
        rows.append({"shape": [B, L, H, D], "query_plus_estimator_us": t_qe, "query_us": t_q, "estimator_us": max(t_qe - t_q, 0.0),
                     "bytes": units * (D // 8 + 4), "paper_hopper_warp_us": warp_ms * 1e3, "paper_hopper_original_us": orig_ms * 1e3})
        for c in caches:
            c.close()
    return {"note": "estimator-only latency beside the paper's Hopper numbers (context, another machine); at these sizes the "
                    "kernels are launch-latency bound", "rows": rows}


def leg_estimator_variants(rb, steps, peak):
    """the estimator at config 2's shape with fp32 factors (20 B/unit), fp16 factors (18 B/unit: the paper's
    2-byte factor, L752) and with query centring (f_bias, +4 G = 16 B/unit; L89); random codes, cold L2 over 8 replicas;
    time = (S3 + S4/S5) - S3."""
    import torch
    B, Hq, Hkv, L, D, R = 1, 32, 8, 131072, 128, 8
    rot = rb.make_rotation(31519, D)
    g = torch.Generator(device="cuda")
    g.manual_seed(6)
    q = torch.randn(B, Hq, D, device="cuda", generator=g).to(torch.bfloat16)
    out = {}
    for name, kw, bpu in (("fp32_factors", {}, 20), ("fp16_factors", dict(factor_dtype=torch.float16), 18),
                          ("fp32_factors_with_cq_f_bias", dict(with_cq=True), 36)):
        caches = []
        for _ in range(R):
            c = rb.RaBitQCache(B, Hq, Hkv, L, rot, head_dim=D, interleave_kv=True, **kw)
            c.codes.copy_(torch.randint(-2 ** 31, 2 ** 31 - 1, c.codes.shape, dtype=torch.int32, device="cuda", generator=g))
            c.f_scale.copy_((torch.rand(c.f_scale.shape, device="cuda", generator=g) + 0.5).to(c.f_scale.dtype))
            if c.f_bias is not None:
                c.f_bias.copy_(torch.randn(c.f_bias.shape, device="cuda", generator=g))
                c.c_q.copy_(torch.randn(c.c_q.shape, device="cuda", generator=g) * 0.1)
            c.n_indexed.fill_(L)
            c.n_total.fill_(L)
            caches.append(c)
        sc = [c.new_scores() for c in caches]
        t_q = ev_time_us(lambda i: caches[i % R].query_quantize(q), steps)
        t_qe = ev_time_us(lambda i: caches[i % R].estimate_scores(q, sc[i % R]), steps)
        est = max(t_qe - t_q, 1e-3)
        byt = B * Hkv * L * bpu
        out[name] = {"bytes_per_unit": bpu, "estimator_us": est, "query_plus_estimator_us": t_qe, "gbs": byt / est / 1e3,
                     "frac_measured": byt / est / 1e3 / peak}
        for c in caches:
            c.close()
        del caches, sc
    return out


def leg_encode(rb, w2, steps):
    """Config 4 (i): index build of 4 x 8 x 131 072 bf16 keys (config 2's keys in every sequence): rbq_encode_keys =
    centroid + Alg.1, canonical fp32 order (EXACT) vs tcgen05 rotation (FAST), dense QR vs Walsh-Hadamard.  Tensor-pipe
    utilisation of the FAST kernel: profiles/ (ncu)."""
    import torch
    from paper_2606_31519_b200 import synth
    B, L = 4, int(w2.seq_lens[0])
    Kb = torch.from_numpy(w2.K[0]).to(torch.bfloat16).cuda()
    seq = torch.full((B,), L, dtype=torch.int32, device="cuda")
    units = B * w2.Hkv * L
    out = {"units": units, "bytes_per_unit": 2 * w2.D + w2.D // 8 + 4}
    for rk, rname in ((rb.RBQ_ROT_DENSE, "dense"), (rb.RBQ_ROT_WH, "wh")):
        rot = rb.make_rotation(31519, w2.D) if rk == rb.RBQ_ROT_DENSE else torch.from_numpy(synth.wh_sign_vector(w2.D))
        for em, ename in ((rb.RBQ_ENC_EXACT, "exact"), (rb.RBQ_ENC_FAST, "fast")):
            c = rb.RaBitQCache(B, w2.Hq, w2.Hkv, w2.Lcap, rot, head_dim=w2.D, rot_kind=rk, enc_mode=em)
            for b in range(B):
                c.K[b].copy_(Kb)
            us = ev_time_us(lambda i: c.encode_keys(seq), max(3, steps // 8), warm=2)
            out[f"{rname}_{ename}"] = {"us": us, "units_per_s": units / us * 1e6, "gbs": units * out["bytes_per_unit"] / us / 1e3}
            c.close()
            del c
    return out


def leg_decode_loop(rb, w, rot, n_steps, label, peak):
    """Configs 3 and 4 (ii): n_steps decode steps, one token per sequence appended per step (rbq_append_tokens, W = 64:
    a batched flush encode every 64 steps), decode step after every append; mean us per (append + step) with the flush on
    the main stream vs on a side stream, and the latency of the flush itself."""
    import torch
    from paper_2606_31519_b200 import synth
    dt = torch.bfloat16
    W = 64
    c = rb.RaBitQCache(w.B, w.Hq, w.Hkv, w.Lcap, rot, head_dim=w.D, kv_dtype=dt, q_dtype=dt, out_dtype=torch.float32, flush_tokens=W)
    c.K.copy_(torch.from_numpy(w.K).to(dt))
    c.V.copy_(torch.from_numpy(w.V).to(dt))
    c.encode_keys(torch.from_numpy(w.seq_lens).cuda())
    pool = [torch.from_numpy(x).to(dt).cuda() for x in synth.query_pool(w, 8)]
    total = 2 * n_steps + 2 * W
    g = torch.Generator(device="cuda")
    g.manual_seed(9)
    new_k = torch.randn(total, w.B, w.Hkv, 1, w.D, device="cuda", generator=g)
    new_k[..., 0:4] *= 10.0
    new_v = torch.randn(total, w.B, w.Hkv, 1, w.D, device="cuda", generator=g)
    new_k, new_v = new_k.to(dt), new_v.to(dt)
    out_t = c.new_out()
    main, side = torch.cuda.current_stream(), torch.cuda.Stream()
    res = {"workload": label, "steps": n_steps, "flush_tokens": W}
    pos = 0
    for name, sd in (("flush_on_main_stream", None), ("flush_on_side_stream", side)):
        for i in range(W):                                  # warm-up, also brings the pending count to a multiple of W
            c.append_tokens(new_k[pos], new_v[pos], stream=main, side_stream=sd)
            c.decode_step(pool[i % 8], w.p, out_t)
            pos += 1
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for i in range(n_steps):
            c.append_tokens(new_k[pos], new_v[pos], stream=main, side_stream=sd)
            c.decode_step(pool[i % 8], w.p, out_t)
            pos += 1
        b.record()
        torch.cuda.synchronize()
        res[name] = {"us_per_step": a.elapsed_time(b) * 1e3 / n_steps}
    # the flush alone: W rows per (sequence, KV head) through rbq_append_tokens in one call on one stream
    kk = new_k[:W].permute(1, 2, 0, 3, 4).reshape(w.B, w.Hkv, W, w.D).contiguous()
    vv = new_v[:W].permute(1, 2, 0, 3, 4).reshape(w.B, w.Hkv, W, w.D).contiguous()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    c.append_tokens(kk, vv)
    b.record()
    torch.cuda.synchronize()
    res["flush_call_us"] = a.elapsed_time(b) * 1e3
    res["flush_units"] = w.B * w.Hkv * W
    # per-stage times (library stage events) and achieved bandwidth of the two streaming kernels at this batch size
    c.profile_enable(True)
    for i in range(16):
        c.decode_step(pool[i % 8], w.p, out_t)
    torch.cuda.synchronize()
    ms, k = c.profile_read()
    c.profile_enable(False)
    st = {key: v * 1e3 / max(1, k) for key, v in ms.items()}
    sel = c.new_sel()
    c.decode_step(pool[0], w.p, out_t, sel[0], sel[1])
    torch.cuda.synchronize()
    n_idx, n_tot = c.n_indexed.cpu().numpy(), c.n_total.cpu().numpy()
    uni, per_head = union_rows(sel[0].cpu().numpy(), sel[1].cpu().numpy(), n_idx, n_tot, w.Hkv)
    est_b = float(n_idx.sum()) * w.Hkv * (w.D // 8 + 4)
    att_b = float(uni) * 2 * w.D * 2
    res["stages_us"] = st
    res["estimator"] = {"bytes": est_b, "gbs": est_b / st["estimator"] / 1e3, "frac_measured": est_b / st["estimator"] / 1e3 / peak}
    res["attn_gather"] = {"bytes": att_b, "gbs": att_b / st["attn_gather"] / 1e3, "frac_measured": att_b / st["attn_gather"] / 1e3 / peak}
    res["budget_mean_tokens"] = float(sel[1].float().mean().item())
    res["overflow_flag"] = c.status_flags()
    c.close()
    return res


def leg_gather4(rb, rot, peak):
    """SURVEY 7 hard part 5 / VERDICT r1 item 5(c): random 256-byte row gathers by 16-byte cp.async (what S7 uses) against TMA
    tile::gather4, on separate K and V matrices and on one matrix of interleaved K | V rows; rbq_diag_gather streams ~462 K
    of 1 M rows (config 2's union density) with the gather kernel's launch shape and pipeline depth, cold L2 over 4 replicas."""
    import torch
    c = rb.RaBitQCache(1, 32, 8, 4096, rot)
    g = torch.Generator(device="cuda")
    g.manual_seed(3)
    n_rows, R = 8 * 131072, 4
    Ks = [torch.randn(n_rows, 128, device="cuda", generator=g).to(torch.bfloat16) for _ in range(R)]
    Vs = [torch.randn(n_rows, 128, device="cuda", generator=g).to(torch.bfloat16) for _ in range(R)]
    rows = torch.nonzero(torch.rand(n_rows, device="cuda", generator=g) < 0.44).flatten().to(torch.int32)
    cs = torch.zeros(1, dtype=torch.int64, device="cuda")
    out = {"rows": int(rows.numel()), "of_rows": n_rows, "bytes": int(rows.numel()) * 512}
    names = {0: "cp_async_separate_kv", 1: "tma_gather4_separate_kv", 2: "cp_async_interleaved_kv", 3: "tma_gather4_interleaved_kv"}
    for mode in (0, 1, 2, 3):
        if mode == 2:
            Ks = [torch.cat([Ks[r], Vs[r]], dim=1).contiguous() for r in range(R)]
            Vs = [None] * R
            torch.cuda.empty_cache()
        us = ev_time_us(lambda i: rb.rbq_diag_gather(c.ctx, Ks[i % R], Vs[i % R], rows, mode, cs), 40)
        out[names[mode]] = {"us": us, "gbs": out["bytes"] / us / 1e3, "frac_measured": out["bytes"] / us / 1e3 / peak}
    c.close()
    return out


def leg_prefill(rb, w1, rot, steps):
    """SURVEY 8(f3) / PAPER.md:L213, L341 (<10 % TTFT overhead): one layer's causal prefill attention (torch SDPA, a library
    call standing in for the model) on the main stream, alone vs with rbq_encode_keys of the same keys on a low-priority
    side stream, joined by an event; config 1's shape (L = 32 768)."""
    import torch
    out = {}
    n = int(w1.seq_lens[0])
    G = w1.Hq // w1.Hkv
    lo, _hi = torch.cuda.Stream.priority_range()
    main, side = torch.cuda.current_stream(), torch.cuda.Stream(priority=lo)
    seq = torch.from_numpy(w1.seq_lens).cuda()
    for em, ename in ((rb.RBQ_ENC_EXACT, "exact"), (rb.RBQ_ENC_FAST, "fast")):
        c = rb.RaBitQCache(w1.B, w1.Hq, w1.Hkv, w1.Lcap, rot, head_dim=w1.D, enc_mode=em)
        c.K.copy_(torch.from_numpy(w1.K).to(torch.bfloat16))
        c.V.copy_(torch.from_numpy(w1.V).to(torch.bfloat16))
        qs = torch.randn(1, w1.Hq, n, w1.D, device="cuda", dtype=torch.bfloat16)
        kk = c.K[:, :, :n].repeat_interleave(G, dim=1).contiguous()
        vv = c.V[:, :, :n].repeat_interleave(G, dim=1).contiguous()

        def attn_only(i):
            torch.nn.functional.scaled_dot_product_attention(qs, kk, vv, is_causal=True)

        def attn_and_index(i):
            side.wait_stream(main)
            torch.nn.functional.scaled_dot_product_attention(qs, kk, vv, is_causal=True)
            c.encode_keys(seq, stream=side)
            main.wait_stream(side)

        reps = max(3, steps // 16)
        t_enc = ev_time_us(lambda i: c.encode_keys(seq), reps, warm=2)
        t_a = ev_time_us(attn_only, reps, warm=2)
        t_b = ev_time_us(attn_and_index, reps, warm=2)
        out[ename] = {"attention_us": t_a, "attention_with_index_build_us": t_b, "index_build_alone_us": t_enc,
                      "overhead_pct": 100.0 * (t_b - t_a) / t_a}
        c.close()
        del c, qs, kk, vv
    out["note"] = "against the attention of ONE layer only (no projections / MLP); the paper's bound is < 10 % of TTFT"
    return out


def leg_recall(w, cache, q_dev, sel_idx, sel_cnt):
    """Attention recall of the selected set under the EXACT softmax (the paper's metric, L280): per head the softmax mass of
    the selected tokens, logits from the true keys (torch matmul on the device: a diagnostic, outside every timed region)."""
    import torch
    G = w.Hq // w.Hkv
    rec = []
    for b in range(w.B):
        n = int(w.seq_lens[b])
        for h in range(w.Hq):
            k = cache.K[b, h // G, :n].float()
            lg = (k @ q_dev[b, h].float()) / math.sqrt(w.D)
            pr = torch.softmax(lg, dim=0)
            idx = torch.as_tensor(np.asarray(sel_idx[b, h, :int(sel_cnt[b, h])]), device=pr.device).long()
            rec.append(float(pr[idx].sum().item()))
    rec = np.array(rec)
    return {"min": float(rec.min()), "mean": float(rec.mean()), "max": float(rec.max())}


def cpu_stage_baseline(w, budget_s=6.0):
    """The oracle per stage (encode, estimate, Top-p, attention) on ONE KV head (G query heads) of the workload, timed at all
    host threads and at 1 thread; times scaled by Hkv to the full step (SURVEY 8(d) "CPU baseline")."""
    from oracle import rbq_oracle as orc
    G = w.Hq // w.Hkv
    K, V, q = np.ascontiguousarray(w.K[:, :1]), np.ascontiguousarray(w.V[:, :1]), np.ascontiguousarray(w.q[:, :G])
    rot, _ = orc.rotation_from_gaussian(w.rot_gauss)
    sm = 1.0 / math.sqrt(w.D)
    nmax = orc.max_threads()
    res = {"sample": f"1 of {w.Hkv} KV heads ({G} query heads), full context, one call per stage, scaled x{w.Hkv}", "unit": "us"}
    for nt in (nmax, 1):
        orc.set_threads(nt)
        t0 = time.perf_counter()
        c_k = orc.centroid(K, w.seq_lens)
        codes, fs, _ = orc.encode(K, np.zeros_like(w.seq_lens), w.seq_lens, orc.ROT_DENSE, rot, c_k)
        t1 = time.perf_counter()
        scores, _, _, _ = orc.estimate_scores(q, codes, fs, None, c_k, None, w.seq_lens, orc.ROT_DENSE, rot, sm)
        t2 = time.perf_counter()
        sel_idx, sel_cnt = orc.topp(scores.reshape(w.B * G, w.Lcap), np.repeat(w.seq_lens, G), w.p)
        t3 = time.perf_counter()
        orc.attention(q, K, V, sel_idx, sel_cnt, w.seq_lens, w.seq_lens, sm)
        t4 = time.perf_counter()
        res[f"threads_{nt}"] = {"encode_setup": (t1 - t0) * 1e6 * w.Hkv, "estimate": (t2 - t1) * 1e6 * w.Hkv,
                                "topp": (t3 - t2) * 1e6 * w.Hkv, "attention": (t4 - t3) * 1e6 * w.Hkv,
                                "step": (t4 - t1) * 1e6 * w.Hkv}
    orc.set_threads(nmax)
    return res


def run_legs(args, rb, w2, rot, peak):
    """All legs; each one guarded."""
    import torch
    legs = {}
    steps = max(20, min(args.steps, 200))

    def guarded(name, fn):
        t0 = time.time()
        try:
            legs[name] = fn()
        except Exception as e:      # a leg never takes the headline down
            legs[name] = {"error": f"{type(e).__name__}: {e}"}
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        log(f"[bench] leg {name}: {time.time() - t0:.1f}s")

    rot64 = None
    guarded("config0", lambda: leg_static_config(rb, 0, [0.9], rot, steps, peak))
    guarded("config1", lambda: leg_static_config(rb, 1, [0.8, 0.9, 0.95], rot, steps, peak))
    guarded("table5", lambda: leg_table5(rb, steps))
    guarded("estimator_variants", lambda: leg_estimator_variants(rb, steps, peak))
    guarded("config4_encode", lambda: leg_encode(rb, w2, steps))
    guarded("prefill_overlap", lambda: leg_prefill(rb, build_workload(1, None), rot, steps))
    guarded("gather4_experiment", lambda: leg_gather4(rb, rot, peak))
    if not args.quick:
        from paper_2606_31519_b200 import synth
        guarded("config3_decode_loop", lambda: leg_decode_loop(
            rb, synth.make_workload(3, extra_cap=512), rot, 128,
            "BASELINE config 3: B=16, contexts U[16384, 65536], 32 q / 8 KV heads, bf16, p=0.9, W=64", peak))
        guarded("config4_decode_loop", lambda: leg_decode_loop(
            rb, synth.make_workload(4, extra_cap=512), rot, 128,
            "BASELINE config 4 (ii): B=4 x 131072, 32 q / 8 KV heads, bf16, p=0.9, W=64", peak))
    return legs


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
    ap.add_argument("--no-legs", dest="legs", action="store_false", help="headline only (skip the SURVEY 8(d) legs under `configs`)")
    ap.add_argument("--quick", action="store_true", help="skip the two decode-loop legs (configs 3 and 4: ~1 min of host-side generation)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
