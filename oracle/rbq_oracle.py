"""ctypes front-end of the CPU ORACLE (oracle/rbq_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares no code with the CUDA
path (paper_2606_31519_b200/csrc, binding.py) and imports nothing from it.

Every function is a thin wrapper over one `rbq_ref_*` C function (argument marshalling only);
the arithmetic, with its PAPER.md citations, lives in rbq_ref.c.  The only logic written here
is (a) the chained convenience `estimate_scores` / `decode_step` (calls in Alg.2 order,
PAPER.md:L159-190) and (b) the lazy-update state machine `LazyIndex` (reading
R14 in DESIGN.md).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rbq_ref.c"
_LIB = _HERE / "librbq_ref.so"
_lib = None

ROT_DENSE, ROT_WH = 0, 1


def build(force: bool = False) -> Path:
    """gcc -O2, no fast-math, no FP contraction (canonical fp32 order, R1)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-fno-fast-math", "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def set_threads(n: int):
    lib().rbq_ref_set_threads(int(n))


def max_threads() -> int:
    return int(lib().rbq_ref_max_threads())


# --- O1 -----------------------------------------------------------------------------------
def rotation_from_gaussian(A: np.ndarray):
    A = np.ascontiguousarray(A, dtype=np.float64)
    D = A.shape[0]
    r32 = np.zeros((D, D), np.float32)
    r64 = np.zeros((D, D), np.float64)
    rc = lib().rbq_ref_rotation_from_gaussian(_p(A, C.c_double), D, _p(r32, C.c_float), _p(r64, C.c_double))
    assert rc == 0
    return r32, r64


def rotation_wh(signs: np.ndarray) -> np.ndarray:
    s = _f32(signs)
    D = s.shape[0]
    r = np.zeros((D, D), np.float32)
    assert lib().rbq_ref_rotation_wh(_p(s, C.c_float), D, _p(r, C.c_float)) == 0
    return r


def fwht(u: np.ndarray) -> np.ndarray:
    u = _f32(u).copy()
    lib().rbq_ref_fwht(_p(u, C.c_float), u.shape[0])
    return u


# --- O2 -----------------------------------------------------------------------------------
def centroid(K: np.ndarray, seq_lens) -> np.ndarray:
    K = _f32(K)
    B, Hkv, Lcap, D = K.shape
    sl = _i32(seq_lens)
    ck = np.zeros((B, Hkv, D), np.float32)
    assert lib().rbq_ref_centroid(_p(K, C.c_float), B, Hkv, Lcap, D, _p(sl, C.c_int32), _p(ck, C.c_float)) == 0
    return ck


def encode(K, t_begin, t_end, rot_kind, rot, c_k, c_q=None, Hq=0, codes=None, f_scale=None, f_bias=None):
    """Alg.1 for tokens [t_begin[b], t_end[b]).  Returns (codes, f_scale, f_bias)."""
    K = _f32(K)
    B, Hkv, Lcap, D = K.shape
    tb, te = _i32(t_begin), _i32(t_end)
    rot, c_k = _f32(rot), _f32(c_k)
    if codes is None:
        codes = np.zeros((B, Hkv, Lcap, D // 32), np.uint32)
    if f_scale is None:
        f_scale = np.zeros((B, Hkv, Lcap), np.float32)
    if c_q is not None:
        c_q = _f32(c_q)
        Hq = c_q.shape[1]
        if f_bias is None:
            f_bias = np.zeros((B, Hq, Lcap), np.float32)
    rc = lib().rbq_ref_encode(_p(K, C.c_float), B, Hkv, Lcap, D, _p(tb, C.c_int32), _p(te, C.c_int32),
                              int(rot_kind), _p(rot, C.c_float), _p(c_k, C.c_float), _p(c_q, C.c_float),
                              int(Hq), _p(codes, C.c_uint32), _p(f_scale, C.c_float), _p(f_bias, C.c_float))
    assert rc == 0
    return codes, f_scale, f_bias


def round_factors_f16(f_scale: np.ndarray) -> np.ndarray:
    """O2c: the stored factors rounded to IEEE binary16 (RNE) and widened back; returns a new array."""
    f = _f32(f_scale).copy()
    fn = lib().rbq_ref_round_factors_f16
    fn.argtypes = [C.c_void_p, C.c_longlong]
    assert fn(f.ctypes.data, f.size) == 0
    return f


# --- O3 -----------------------------------------------------------------------------------
def query_prep(q, Hkv, rot_kind, rot, c_k, c_q=None):
    q = _f32(q)
    B, Hq, D = q.shape
    rot, c_k = _f32(rot), _f32(c_k)
    c_q = None if c_q is None else _f32(c_q)
    out = dict(qu=np.zeros((B, Hq, D), np.uint8), qn=np.zeros((B, Hq), np.float32),
               ql=np.zeros((B, Hq), np.float32), delta=np.zeros((B, Hq), np.float32),
               sumq=np.zeros((B, Hq), np.int32), q_ck=np.zeros((B, Hq), np.float32),
               cq_ck=np.zeros((B, Hq), np.float32), qprime=np.zeros((B, Hq, D), np.float32))
    rc = lib().rbq_ref_query_prep(_p(q, C.c_float), B, Hq, Hkv, D, int(rot_kind), _p(rot, C.c_float),
                                  _p(c_q, C.c_float), _p(c_k, C.c_float), _p(out["qu"], C.c_uint8),
                                  _p(out["qn"], C.c_float), _p(out["ql"], C.c_float),
                                  _p(out["delta"], C.c_float), _p(out["sumq"], C.c_int32),
                                  _p(out["q_ck"], C.c_float), _p(out["cq_ck"], C.c_float),
                                  _p(out["qprime"], C.c_float))
    assert rc == 0
    return out


# --- O4 -----------------------------------------------------------------------------------
def int_dots(codes, qu, n_indexed, packed=False):
    codes = np.ascontiguousarray(codes, dtype=np.uint32)
    qu = np.ascontiguousarray(qu, dtype=np.uint8)
    B, Hkv, Lcap, W = codes.shape
    Hq, D = qu.shape[1], qu.shape[2]
    ni = _i32(n_indexed)
    dot = np.zeros((B, Hq, Lcap), np.int32)
    pop = np.zeros((B, Hkv, Lcap), np.int32)
    fn = lib().rbq_ref_int_dots_packed if packed else lib().rbq_ref_int_dots
    rc = fn(_p(codes, C.c_uint32), _p(qu, C.c_uint8), B, Hq, Hkv, Lcap, D, _p(ni, C.c_int32),
            _p(dot, C.c_int32), _p(pop, C.c_int32))
    assert rc == 0
    return dot, pop


# --- O5 -----------------------------------------------------------------------------------
def logits(dot, pop, f_scale, f_bias, qp, n_indexed, sm_scale, D):
    dot = _i32(dot)
    pop = _i32(pop)
    B, Hq, Lcap = dot.shape
    Hkv = pop.shape[1]
    f_scale = _f32(f_scale)
    f_bias = None if f_bias is None else _f32(f_bias)
    ni = _i32(n_indexed)
    scores = np.zeros((B, Hq, Lcap), np.float32)
    fn = lib().rbq_ref_logits
    fn.argtypes = [C.c_void_p] * 10 + [C.c_int] * 5 + [C.c_void_p, C.c_double, C.c_void_p]
    rc = fn(dot.ctypes.data, pop.ctypes.data, f_scale.ctypes.data,
            None if f_bias is None else f_bias.ctypes.data,
            _f32(qp["qn"]).ctypes.data, _f32(qp["ql"]).ctypes.data, _f32(qp["delta"]).ctypes.data,
            _i32(qp["sumq"]).ctypes.data, _f32(qp["q_ck"]).ctypes.data, _f32(qp["cq_ck"]).ctypes.data,
            B, Hq, Hkv, Lcap, D, ni.ctypes.data, float(sm_scale), scores.ctypes.data)
    assert rc == 0
    return scores


def estimate_scores(q, codes, f_scale, f_bias, c_k, c_q, n_indexed, rot_kind, rot, sm_scale):
    """Alg.2 steps 1-2 chained: O3 -> O4 -> O5."""
    Hkv, D = codes.shape[1], q.shape[2]
    qp = query_prep(q, Hkv, rot_kind, rot, c_k, c_q)
    dot, pop = int_dots(codes, qp["qu"], n_indexed)
    return logits(dot, pop, f_scale, f_bias, qp, n_indexed, sm_scale, D), qp, dot, pop


# --- O6 -----------------------------------------------------------------------------------
def topp(scores, n_per_row, p):
    """scores [rows][Lcap]; returns (sel_idx [rows][Lcap] in (prob desc, idx asc) order, sel_cnt)."""
    scores = _f32(scores)
    rows, Lcap = scores.shape
    n = _i32(n_per_row)
    sel_idx = np.full((rows, Lcap), -1, np.int32)
    sel_cnt = np.zeros(rows, np.int32)
    fn = lib().rbq_ref_topp
    fn.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
    rc = fn(scores.ctypes.data, rows, Lcap, n.ctypes.data, float(p), sel_idx.ctypes.data, sel_cnt.ctypes.data)
    assert rc == 0
    return sel_idx, sel_cnt


def topp_alg3(prob, p):
    prob = np.ascontiguousarray(prob, dtype=np.float64)
    mask = np.zeros(prob.shape[0], np.uint8)
    fn = lib().rbq_ref_topp_alg3
    fn.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_void_p]
    it = fn(prob.ctypes.data, prob.shape[0], float(p), mask.ctypes.data)
    return mask.astype(bool), it


# --- O7 -----------------------------------------------------------------------------------
def attention(q, K, V, sel_idx, sel_cnt, n_indexed, n_total, sm_scale):
    q, K, V = _f32(q), _f32(K), _f32(V)
    B, Hq, D = q.shape
    Hkv, Lcap = K.shape[1], K.shape[2]
    sel_idx = _i32(sel_idx).reshape(B, Hq, Lcap)
    sel_cnt = _i32(sel_cnt).reshape(B, Hq)
    ni, nt = _i32(n_indexed), _i32(n_total)
    out = np.zeros((B, Hq, D), np.float32)
    lse = np.zeros((B, Hq), np.float32)
    fn = lib().rbq_ref_attention
    fn.argtypes = [C.c_void_p] * 3 + [C.c_int] * 5 + [C.c_void_p] * 4 + [C.c_double, C.c_void_p, C.c_void_p]
    rc = fn(q.ctypes.data, K.ctypes.data, V.ctypes.data, B, Hq, Hkv, Lcap, D, sel_idx.ctypes.data,
            sel_cnt.ctypes.data, ni.ctypes.data, nt.ctypes.data, float(sm_scale), out.ctypes.data,
            lse.ctypes.data)
    assert rc == 0
    return out, lse


def decode_step(q, K, V, codes, f_scale, f_bias, c_k, c_q, n_indexed, n_total, rot_kind, rot, p, sm_scale):
    """Alg.2 end to end: estimate -> Top-p over indexed tokens -> attention
    over selected U pending."""
    B, Hq, D = q.shape
    Lcap = codes.shape[2]
    scores, _, _, _ = estimate_scores(q, codes, f_scale, f_bias, c_k, c_q, n_indexed, rot_kind, rot, sm_scale)
    n_rows = np.repeat(_i32(n_indexed), Hq)
    sel_idx, sel_cnt = topp(scores.reshape(B * Hq, Lcap), n_rows, p)
    out, lse = attention(q, K, V, sel_idx, sel_cnt, n_indexed, n_total, sm_scale)
    return dict(out=out, lse=lse, scores=scores, sel_idx=sel_idx.reshape(B, Hq, Lcap),
                sel_cnt=sel_cnt.reshape(B, Hq))


# --- O8 lazy updates (reading R14) -------------------------------------
class LazyIndex:
    """State machine of the lazy decode update: new rows go to the full-precision tail; when
    the number of pending rows reaches W, the oldest floor(pending/W)*W pending rows are encoded in
    one batch with the frozen c_k; they stay pending (attended exactly, excluded from Top-p) until
    the NEXT append call commits them (n_indexed += flushed)."""

    def __init__(self, K, V, seq_lens, rot_kind, rot, W, c_q=None, factor_f16=False):
        self.K, self.V = _f32(K).copy(), _f32(V).copy()
        self.rot_kind, self.rot, self.W, self.c_q = rot_kind, _f32(rot), int(W), c_q
        self.factor_f16 = factor_f16
        sl = _i32(seq_lens)
        self.c_k = centroid(self.K, sl)
        self.codes, self.f_scale, self.f_bias = encode(self.K, np.zeros_like(sl), sl, rot_kind, self.rot,
                                                       self.c_k, c_q)
        if factor_f16:
            self.f_scale = round_factors_f16(self.f_scale)
        self.n_indexed = sl.copy()
        self.n_total = sl.copy()
        self.in_flight = 0

    def append(self, k_new, v_new):
        if self.in_flight:                       # commit the flush enqueued by the previous call
            self.n_indexed = self.n_indexed + self.in_flight
            self.in_flight = 0
        n_new = k_new.shape[2]
        for b in range(self.K.shape[0]):
            t0 = int(self.n_total[b])
            self.K[b, :, t0:t0 + n_new] = k_new[b]
            self.V[b, :, t0:t0 + n_new] = v_new[b]
        self.n_total = self.n_total + n_new
        pending = int(self.n_total[0] - self.n_indexed[0])
        if self.W > 0 and pending >= self.W:
            nf = pending // self.W * self.W
            encode(self.K, self.n_indexed, self.n_indexed + nf, self.rot_kind, self.rot, self.c_k, self.c_q,
                   codes=self.codes, f_scale=self.f_scale, f_bias=self.f_bias)
            if self.factor_f16:       # idempotent on the already rounded prefix
                self.f_scale = round_factors_f16(self.f_scale)
            self.in_flight = nf
