"""Seeded synthetic workloads for the RaBitQCache decode hot path.

This module only DRAWS INPUTS (keys, values, queries, Gaussian matrices, sign vectors,
sequence lengths).  It contains none of the method's arithmetic (no rotation, no
encoding, no estimator, no Top-p, no attention): both the CUDA path and the CPU oracle
consume the arrays it returns, and neither is imported here.  Pure numpy.

Recipe: SURVEY.md section 8(d) / DESIGN.md section 4, shapes from BASELINE.json `configs`.
The paper measured on LongBench / RULER / GSM8K prompts with Llama / Longchat weights
(PAPER.md:L299, L339); none of that is available, so these inputs stand in for them:
Llama-3.1-8B attention geometry, outlier channels, attention sinks, a few heavy tokens,
per-head sparsity spread calibrated so that Top-p budgets land in the paper's 4-25 % range
(PAPER.md:L846, L869, L930-936).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED = 31519
D_HEAD = 128
N_SINK = 4
SINK_MASS = 0.3


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest bfloat16 (ties to even), returned as float32."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    u = (u + r) & np.uint32(0xFFFF0000)
    return u.view(np.float32)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 values that are bf16-representable -> their 16-bit patterns (uint16)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return (u >> 16).astype(np.uint16)


@dataclass
class Workload:
    cfg: int
    variant: str
    B: int
    Hq: int
    Hkv: int
    D: int
    Lcap: int
    seq_lens: np.ndarray          # int32 [B]
    kv_dtype: str                 # "f32" | "bf16"
    K: np.ndarray                 # float32 [B][Hkv][Lcap][D] (bf16-representable when bf16)
    V: np.ndarray
    q: np.ndarray                 # float32 [B][Hq][D]
    c_q: np.ndarray | None        # float32 [B][Hq][D] or None
    p: float
    flush_tokens: int
    rot_gauss: np.ndarray         # float64 [D][D] Gaussian matrix (input of the QR rotation)
    wh_signs: np.ndarray          # float32 [D] in {-1,+1}
    sigma: np.ndarray = field(default=None)   # float64 [B][Hq] target bulk-logit std

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv


def rotation_gaussian(D: int = D_HEAD) -> np.ndarray:
    return np.random.default_rng([SEED, 99]).standard_normal((D, D))


def wh_sign_vector(D: int = D_HEAD) -> np.ndarray:
    return (np.random.default_rng([SEED, 98]).integers(0, 2, D) * 2 - 1).astype(np.float32)


_CFG = {
    # cfg: (B, Hq, Hkv, L, dtype, n_heavy, knob, p, W)
    0: (1, 1, 1, 4096, "f32", 16, "fixed", 0.9, 0),
    1: (1, 32, 8, 32768, "bf16", 64, "spread", 0.9, 0),
    2: (1, 32, 8, 131072, "bf16", 256, "temp", 0.9, 0),
    3: (16, 32, 8, None, "bf16", 64, "spread", 0.9, 64),
    4: (4, 32, 8, 131072, "bf16", 256, "temp", 0.9, 64),
}


def config_seq_lens(cfg: int, B: int | None = None, L: int | None = None) -> np.ndarray:
    b0, _, _, l0, *_ = _CFG[cfg]
    B = b0 if B is None else B
    if L is not None:
        if cfg == 3:   # keep the ragged mix, scaled to [L/4, L]
            return np.random.default_rng([SEED, 3]).integers(max(8, L // 4), L + 1, B).astype(np.int32)
        return np.full(B, L, np.int32)
    if cfg == 3:
        return np.random.default_rng([SEED, 3]).integers(16384, 65537, B).astype(np.int32)
    return np.full(B, l0, np.int32)


def _draw_group(cfg, b, g, L, G, n_heavy, knob, variant, dtype, D=D_HEAD):
    """One (sequence, KV head): keys, values and the G queries that read them."""
    rng = np.random.default_rng([SEED, cfg, b, g] if D == D_HEAD else [SEED, cfg, b, g, D])
    K = rng.standard_normal((L, D), dtype=np.float32)
    K[:, 0:4] *= 10.0
    V = rng.standard_normal((L, D), dtype=np.float32)
    V[:, 0:4] *= 10.0
    qs = np.zeros((G, D), np.float64)
    sig = np.zeros(G)
    n_heavy = min(n_heavy, max(1, (L - N_SINK) // 2))
    for j in range(G):
        H = N_SINK + rng.choice(L - N_SINK, n_heavy, replace=False)
        m = K[H].astype(np.float64).mean(axis=0)
        q0 = 3.0 * math.sqrt(D) * m / np.linalg.norm(m) + rng.standard_normal(D)
        if knob == "fixed":
            s = 3.0
        elif knob == "spread":
            w = int(rng.integers(8, 513))
            s = 4.0 - (math.log2(w) - 3.0) / 3.0
        else:
            T = float(rng.uniform(0.5, 2.0))
            s = 3.0 / T
        sig[j] = s
        if variant == "C":
            raw = (K[N_SINK:].astype(np.float64) @ q0) / math.sqrt(D)
            q0 = q0 * (s / raw.std())
        qs[j] = q0
    # attention sinks
    if variant == "C":
        n_s = N_SINK if G == 1 else 1
        for j in range(G):
            lg = (K[N_SINK:].astype(np.float64) @ qs[j]) / math.sqrt(D)
            mx = lg.max()
            lse = mx + math.log(np.exp(lg - mx).sum())
            gam = math.sqrt(D) * (math.log(SINK_MASS / (1 - SINK_MASS)) - math.log(n_s) + lse) / (qs[j] @ qs[j])
            if G == 1:
                K[0:N_SINK] = (gam * qs[0]).astype(np.float32)
            elif j < N_SINK:
                K[j] = (gam * qs[j]).astype(np.float32)
    else:  # literal BASELINE.json wording: sink keys = 2 x query
        if G == 1:
            K[0:N_SINK] = (2.0 * qs[0]).astype(np.float32)
        else:
            for j in range(min(G, N_SINK)):
                K[j] = (2.0 * qs[j]).astype(np.float32)
    q32 = qs.astype(np.float32)
    if dtype == "bf16":
        K, V, q32 = bf16_round(K), bf16_round(V), bf16_round(q32)
    return K, V, q32, sig


def make_workload(cfg: int, *, L: int | None = None, B: int | None = None, variant: str = "C",
                  with_cq: bool = False, p: float | None = None, extra_cap: int = 0,
                  n_heavy: int | None = None, D: int = D_HEAD, Hq: int | None = None, Hkv: int | None = None) -> Workload:
    """Build configuration `cfg` of BASELINE.json (optionally scaled down via L / B).

    variant "C" = calibrated (temperature beta, sink gain gamma), "L" = literal wording
    (beta = 1, sink keys = 2 x query; degenerate, parity-only).  `extra_cap` adds room at
    the tail of every sequence for appended tokens.
    """
    b0, Hq0, Hkv0, _, dtype, nh0, knob, p0, W = _CFG[cfg]
    Hq, Hkv = Hq0 if Hq is None else Hq, Hkv0 if Hkv is None else Hkv     # head counts / head_dim other than the config's: SURVEY 8(f1)
    n_heavy = nh0 if n_heavy is None else n_heavy
    seq_lens = config_seq_lens(cfg, B, L)
    B = len(seq_lens)
    G = Hq // Hkv
    Lcap = int(seq_lens.max()) + int(extra_cap)
    Lcap = (Lcap + 63) // 64 * 64
    K = np.zeros((B, Hkv, Lcap, D), np.float32)
    V = np.zeros((B, Hkv, Lcap, D), np.float32)
    q = np.zeros((B, Hq, D), np.float32)
    sigma = np.zeros((B, Hq))
    for b in range(B):
        Lb = int(seq_lens[b])
        for g in range(Hkv):
            k_, v_, q_, s_ = _draw_group(cfg, b, g, Lb, G, n_heavy, knob, variant, dtype, D)
            K[b, g, :Lb], V[b, g, :Lb] = k_, v_
            q[b, g * G:(g + 1) * G] = q_
            sigma[b, g * G:(g + 1) * G] = s_
    c_q = None
    if with_cq:
        c_q = (0.5 * np.random.default_rng([SEED, cfg, 97]).standard_normal((B, Hq, D))).astype(np.float32)
    return Workload(cfg=cfg, variant=variant, B=B, Hq=Hq, Hkv=Hkv, D=D, Lcap=Lcap, seq_lens=seq_lens,
                    kv_dtype=dtype, K=K, V=V, q=q, c_q=c_q, p=p0 if p is None else p, flush_tokens=W,
                    rot_gauss=rotation_gaussian(D), wh_signs=wh_sign_vector(D), sigma=sigma)


def append_rows(cfg: int, step: int, B: int, Hkv: int, n_new: int, dtype: str = "bf16", D: int = D_HEAD):
    """Plain K, V rows for tokens appended at decode step `step` (drawn as recipe step 1)."""
    rng = np.random.default_rng([SEED, cfg, 1000 + step])
    K = rng.standard_normal((B, Hkv, n_new, D), dtype=np.float32)
    K[..., 0:4] *= 10.0
    V = rng.standard_normal((B, Hkv, n_new, D), dtype=np.float32)
    V[..., 0:4] *= 10.0
    if dtype == "bf16":
        K, V = bf16_round(K), bf16_round(V)
    return K, V


def query_pool(w: Workload, n_sets: int = 8) -> np.ndarray:
    """A pool of `n_sets` query sets per sequence, cycled across decode steps (config 3/4):
    set 0 is the workload's own calibrated query; set i > 0 perturbs it with seeded Gaussian
    noise of 25 % of its RMS, re-rounded to the workload dtype (different heavy mixes)."""
    out = np.zeros((n_sets,) + w.q.shape, np.float32)
    out[0] = w.q
    rms = np.sqrt((w.q.astype(np.float64) ** 2).mean(axis=-1, keepdims=True))
    for i in range(1, n_sets):
        rng = np.random.default_rng([SEED, w.cfg, 500 + i])
        x = w.q + (0.25 * rms * rng.standard_normal(w.q.shape)).astype(np.float32)
        out[i] = bf16_round(x) if w.kv_dtype == "bf16" else x
    return out
