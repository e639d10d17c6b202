"""Thin ctypes binding of librbq_b200.so (include/rbq.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels.  PyTorch is used for device memory and streams, nothing else.

There is NO CPU fallback: if the shared library is missing or no CUDA device is present, every
entry point raises.

Function names mirror the C ABI: rbq_create, rbq_encode_keys, rbq_append_tokens, rbq_query_quantize,
rbq_int4_dot_binary, rbq_estimate_scores, rbq_topp_select, rbq_sparse_attention, rbq_decode_step,
rbq_decode_step_host.  `RaBitQCache` bundles a context, its workspace, a K/V cache and an index.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

import os

_HERE = Path(__file__).resolve().parent
# RBQ_B200_LIB selects another build of the same library (the -DRBQ_PROBE build for in-kernel timelines)
LIB_PATH = Path(os.environ["RBQ_B200_LIB"]) if os.environ.get("RBQ_B200_LIB") else _HERE / "librbq_b200.so"
_lib = None

RBQ_F32, RBQ_BF16, RBQ_F16 = 0, 1, 2
RBQ_ROT_DENSE, RBQ_ROT_WH = 0, 1
RBQ_ENC_EXACT, RBQ_ENC_FAST = 0, 1
RBQ_CK_GIVEN = 1

EXPORTS = ["rbq_create", "rbq_destroy", "rbq_workspace_bytes", "rbq_set_workspace", "rbq_last_error",
           "rbq_launch_count", "rbq_encode_keys", "rbq_append_tokens", "rbq_query_quantize",
           "rbq_int4_dot_binary", "rbq_estimate_scores", "rbq_topp_select", "rbq_topp_select_static", "rbq_topp_select_alg3", "rbq_sparse_attention",
           "rbq_decode_step", "rbq_decode_step_host", "rbq_profile_enable", "rbq_profile_read", "rbq_status_flags", "rbq_probe_dump", "rbq_diag_gather"]
N_STAGES = 5
STAGE_NAMES = ["query_prep", "estimator", "topp", "attn_plan", "attn_gather"]


class RbqError(RuntimeError):
    pass


class rbq_config(C.Structure):
    _fields_ = [("batch", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("max_tokens", C.c_int32), ("flush_tokens", C.c_int32), ("kv_dtype", C.c_int32),
                ("q_dtype", C.c_int32), ("out_dtype", C.c_int32), ("sm_scale", C.c_float), ("rot_kind", C.c_int32),
                ("rot", C.c_void_p), ("enc_mode", C.c_int32), ("factor_dtype", C.c_int32)]


class rbq_kv(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("stride_b", C.c_int64), ("stride_h", C.c_int64),
                ("stride_t", C.c_int64)]


class rbq_index(C.Structure):
    _fields_ = [("codes", C.c_void_p), ("f_scale", C.c_void_p), ("f_bias", C.c_void_p), ("c_k", C.c_void_p),
                ("c_q", C.c_void_p), ("n_indexed", C.c_void_p), ("n_total", C.c_void_p)]


def load():
    """Load librbq_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RbqError(f"{LIB_PATH} not found: build it with `python -m paper_2606_31519_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    vp, i32, u32, f32 = C.c_void_p, C.c_int32, C.c_uint32, C.c_float
    sig = {
        "rbq_create": ([C.POINTER(rbq_config), C.POINTER(vp)], C.c_int),
        "rbq_destroy": ([vp], C.c_int),
        "rbq_workspace_bytes": ([vp, C.POINTER(C.c_size_t)], C.c_int),
        "rbq_set_workspace": ([vp, vp, C.c_size_t], C.c_int),
        "rbq_last_error": ([vp], C.c_char_p),
        "rbq_launch_count": ([vp], C.c_int64),
        "rbq_encode_keys": ([vp, C.POINTER(rbq_kv), vp, u32, C.POINTER(rbq_index), vp], C.c_int),
        "rbq_append_tokens": ([vp, vp, vp, i32, C.POINTER(rbq_kv), C.POINTER(rbq_index), vp, vp], C.c_int),
        "rbq_query_quantize": ([vp, vp, C.POINTER(rbq_index), vp, vp, vp], C.c_int),
        "rbq_int4_dot_binary": ([vp, vp, C.POINTER(rbq_index), vp, vp, vp], C.c_int),
        "rbq_estimate_scores": ([vp, vp, C.POINTER(rbq_index), vp, vp], C.c_int),
        "rbq_topp_select": ([vp, vp, C.POINTER(rbq_index), f32, vp, vp, vp], C.c_int),
        "rbq_topp_select_static": ([vp, vp, C.POINTER(rbq_index), f32, vp, vp, vp], C.c_int),
        "rbq_topp_select_alg3": ([vp, vp, C.POINTER(rbq_index), f32, vp, vp, vp, vp], C.c_int),
        "rbq_sparse_attention": ([vp, vp, C.POINTER(rbq_kv), C.POINTER(rbq_index), vp, vp, vp, vp, vp], C.c_int),
        "rbq_decode_step": ([vp, vp, C.POINTER(rbq_kv), C.POINTER(rbq_index), f32, vp, vp, vp, vp], C.c_int),
        "rbq_decode_step_host": ([vp, vp, C.POINTER(rbq_kv), C.POINTER(rbq_index), f32, vp, vp], C.c_int),
        "rbq_profile_enable": ([vp, C.c_int], C.c_int),
        "rbq_profile_read": ([vp, C.POINTER(C.c_float), C.POINTER(i32)], C.c_int),
        "rbq_status_flags": ([vp, C.POINTER(u32), vp], C.c_int),
        "rbq_probe_dump": ([vp, C.c_int, vp], C.c_int),
        "rbq_diag_gather": ([vp, vp, vp, C.c_longlong, vp, C.c_longlong, C.c_int, vp, vp], C.c_int),
    }
    for name, (args, res) in sig.items():
        fn = getattr(lib, name)
        fn.argtypes, fn.restype = args, res
    _lib = lib
    return lib


def _dt(t: torch.dtype) -> int:
    if t == torch.float32:
        return RBQ_F32
    if t == torch.bfloat16:
        return RBQ_BF16
    raise RbqError(f"unsupported dtype {t}")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(s):
    if s is None:
        s = torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream if hasattr(s, "cuda_stream") else int(s))


def _check(ctx, rc, what):
    if rc != 0:
        msg = load().rbq_last_error(ctx).decode() if ctx else ""
        raise RbqError(f"{what} failed with status {rc}: {msg}")


def make_rotation(seed: int, D: int = 128) -> torch.Tensor:
    """A Haar-distributed orthogonal P (QR of a seeded Gaussian matrix, positive-diagonal factor),
    generated once at initialisation with numpy on the host; float32 [D][D]."""
    A = np.random.default_rng(seed).standard_normal((D, D))
    Q, R = np.linalg.qr(A)
    return torch.from_numpy((Q * np.sign(np.diag(R))).astype(np.float32))


# ---- raw entry points (same names as the C ABI) ----------------------------------------------------
def rbq_create(cfg: rbq_config):
    if not torch.cuda.is_available():
        raise RbqError("no CUDA device: the RaBitQCache path has no CPU fallback")
    h = C.c_void_p()
    _check(None, load().rbq_create(C.byref(cfg), C.byref(h)), "rbq_create")
    return h


def rbq_destroy(ctx):
    load().rbq_destroy(ctx)


def rbq_workspace_bytes(ctx) -> int:
    n = C.c_size_t()
    _check(ctx, load().rbq_workspace_bytes(ctx, C.byref(n)), "rbq_workspace_bytes")
    return n.value


def rbq_set_workspace(ctx, ws: torch.Tensor):
    _check(ctx, load().rbq_set_workspace(ctx, _ptr(ws), ws.numel() * ws.element_size()), "rbq_set_workspace")


def rbq_launch_count(ctx) -> int:
    return int(load().rbq_launch_count(ctx))


def rbq_encode_keys(ctx, kv: rbq_kv, seq_lens, flags, idx: rbq_index, stream=None):
    _check(ctx, load().rbq_encode_keys(ctx, C.byref(kv), _ptr(seq_lens), flags, C.byref(idx), _stream(stream)),
           "rbq_encode_keys")


def rbq_append_tokens(ctx, k_new, v_new, n_new, kv: rbq_kv, idx: rbq_index, stream=None, side_stream=None):
    s = _stream(stream)
    _check(ctx, load().rbq_append_tokens(ctx, _ptr(k_new), _ptr(v_new), n_new, C.byref(kv), C.byref(idx), s,
                                         s if side_stream is None else _stream(side_stream)), "rbq_append_tokens")


def rbq_query_quantize(ctx, q, idx: rbq_index, qu=None, qparams=None, stream=None):
    _check(ctx, load().rbq_query_quantize(ctx, _ptr(q), C.byref(idx), _ptr(qu), _ptr(qparams), _stream(stream)),
           "rbq_query_quantize")


def rbq_int4_dot_binary(ctx, q, idx: rbq_index, dot, pop, stream=None):
    _check(ctx, load().rbq_int4_dot_binary(ctx, _ptr(q), C.byref(idx), _ptr(dot), _ptr(pop), _stream(stream)),
           "rbq_int4_dot_binary")


def rbq_estimate_scores(ctx, q, idx: rbq_index, scores, stream=None):
    _check(ctx, load().rbq_estimate_scores(ctx, _ptr(q), C.byref(idx), _ptr(scores), _stream(stream)),
           "rbq_estimate_scores")


def rbq_topp_select(ctx, scores, idx: rbq_index, p, sel_idx, sel_cnt, stream=None):
    _check(ctx, load().rbq_topp_select(ctx, _ptr(scores), C.byref(idx), float(p), _ptr(sel_idx), _ptr(sel_cnt),
                                       _stream(stream)), "rbq_topp_select")


def rbq_topp_select_static(ctx, scores, idx: rbq_index, p, sel_idx, sel_cnt, stream=None):
    """rbq_topp_select without workspace or allocation: scratch in the library's static 2 MiB device array (rbq.h)."""
    _check(ctx, load().rbq_topp_select_static(ctx, _ptr(scores), C.byref(idx), float(p), _ptr(sel_idx), _ptr(sel_cnt),
                                              _stream(stream)), "rbq_topp_select_static")


def rbq_topp_select_alg3(ctx, scores, idx: rbq_index, p, sel_idx, sel_cnt, iters=None, stream=None):
    _check(ctx, load().rbq_topp_select_alg3(ctx, _ptr(scores), C.byref(idx), float(p), _ptr(sel_idx), _ptr(sel_cnt),
                                            _ptr(iters), _stream(stream)), "rbq_topp_select_alg3")


def rbq_sparse_attention(ctx, q, kv: rbq_kv, idx: rbq_index, sel_idx, sel_cnt, out, lse=None, stream=None):
    _check(ctx, load().rbq_sparse_attention(ctx, _ptr(q), C.byref(kv), C.byref(idx), _ptr(sel_idx), _ptr(sel_cnt),
                                            _ptr(out), _ptr(lse), _stream(stream)), "rbq_sparse_attention")


def rbq_decode_step(ctx, q, kv: rbq_kv, idx: rbq_index, p, out, sel_idx=None, sel_cnt=None, stream=None):
    _check(ctx, load().rbq_decode_step(ctx, _ptr(q), C.byref(kv), C.byref(idx), float(p), _ptr(out), _ptr(sel_idx),
                                       _ptr(sel_cnt), _stream(stream)), "rbq_decode_step")


def rbq_decode_step_host(ctx, q_host, kv: rbq_kv, idx: rbq_index, p, out_host, stream=None):
    _check(ctx, load().rbq_decode_step_host(ctx, _ptr(q_host), C.byref(kv), C.byref(idx), float(p), _ptr(out_host),
                                            _stream(stream)), "rbq_decode_step_host")


def rbq_profile_enable(ctx, enable: bool):
    _check(ctx, load().rbq_profile_enable(ctx, int(bool(enable))), "rbq_profile_enable")


def rbq_profile_read(ctx):
    """Blocks until the recorded steps finished; returns ({stage: total ms}, n_steps)."""
    ms = (C.c_float * N_STAGES)()
    n = C.c_int32()
    _check(ctx, load().rbq_profile_read(ctx, ms, C.byref(n)), "rbq_profile_read")
    return dict(zip(STAGE_NAMES, [float(x) for x in ms])), n.value


def rbq_probe_dump(ctx, kernel: int) -> np.ndarray:
    """Probe build only (RBQ_B200_LIB=.../librbq_b200_probe.so): uint64 [256 CTAs][16 slots] of clock64 stamps."""
    out = np.zeros((256, 16), np.uint64)
    _check(ctx, load().rbq_probe_dump(ctx, int(kernel), out.ctypes.data_as(C.c_void_p)), "rbq_probe_dump")
    return out


def rbq_diag_gather(ctx, K, V, rows, mode: int, checksum, stream=None) -> None:
    """Row-gather experiment (rbq.h): modes 0 / 1: K, V bf16 [n_rows_total][128] contiguous; modes 2 / 3: K = interleaved
    K | V rows, bf16 [n_rows_total][256], V = None.  rows int32 [n], checksum int64 [1] (added to).  Even modes: cp.async
    staging, odd modes: TMA tile::gather4."""
    width = 128 if mode < 2 else 256
    assert K.dtype == torch.bfloat16 and K.is_contiguous() and K.shape[-1] == width
    assert rows.dtype == torch.int32 and checksum.dtype == torch.int64
    if mode < 2:
        assert V.dtype == torch.bfloat16 and V.is_contiguous() and V.shape == K.shape
    n_total = K.numel() // width
    _check(ctx, load().rbq_diag_gather(ctx, _ptr(K), _ptr(V) if mode < 2 else None, n_total, _ptr(rows), rows.numel(), int(mode),
                                       _ptr(checksum), _stream(stream)), "rbq_diag_gather")


def rbq_status_flags(ctx, stream=None) -> int:
    """Blocks: the sticky device status word (RBQ_FLAG_APPEND_OVERFLOW = 1)."""
    f = C.c_uint32()
    _check(ctx, load().rbq_status_flags(ctx, C.byref(f), _stream(stream)), "rbq_status_flags")
    return int(f.value)


# ---- convenience bundle ----------------------------------------------------------------------------
class RaBitQCache:
    """Context + workspace + caller-owned tensors (K/V cache, index) for one attention layer."""

    def __init__(self, batch, n_q_heads, n_kv_heads, max_tokens, rot: torch.Tensor, *, head_dim=128, flush_tokens=0,
                 kv_dtype=torch.bfloat16, q_dtype=None, out_dtype=None, sm_scale=0.0, rot_kind=RBQ_ROT_DENSE,
                 enc_mode=RBQ_ENC_EXACT, with_cq=False, device="cuda", interleave_kv=True, factor_dtype=torch.float32):
        self.dev = torch.device(device)
        self.B, self.Hq, self.Hkv, self.D, self.Lcap = batch, n_q_heads, n_kv_heads, head_dim, max_tokens
        self.kv_dtype = kv_dtype
        self.q_dtype = q_dtype or kv_dtype
        self.out_dtype = out_dtype or torch.float32
        self.rot = rot.to(self.dev, torch.float32).contiguous()
        self.cfg = rbq_config(batch, n_q_heads, n_kv_heads, head_dim, max_tokens, flush_tokens, _dt(kv_dtype),
                              _dt(self.q_dtype), _dt(self.out_dtype), float(sm_scale), rot_kind,
                              self.rot.data_ptr(), enc_mode, RBQ_F16 if factor_dtype == torch.float16 else RBQ_F32)
        self.ctx = rbq_create(self.cfg)
        self.ws = torch.empty(rbq_workspace_bytes(self.ctx), dtype=torch.uint8, device=self.dev)
        rbq_set_workspace(self.ctx, self.ws)
        z = dict(device=self.dev)
        if interleave_kv:
            # one allocation [B][Hkv][Lcap][2][D]: the K row and the V row of a token are adjacent in HBM, so the gather
            # attention fetches 4*D contiguous bytes per attended token (rbq_kv carries the strides: stride_t = 2*D)
            self.KV = torch.zeros(batch, n_kv_heads, max_tokens, 2, head_dim, dtype=kv_dtype, **z)
            self.K, self.V = self.KV[:, :, :, 0, :], self.KV[:, :, :, 1, :]
        else:
            self.K = torch.zeros(batch, n_kv_heads, max_tokens, head_dim, dtype=kv_dtype, **z)
            self.V = torch.zeros(batch, n_kv_heads, max_tokens, head_dim, dtype=kv_dtype, **z)
        self.codes = torch.zeros(batch, n_kv_heads, max_tokens, head_dim // 32, dtype=torch.int32, **z)
        self.f_scale = torch.zeros(batch, n_kv_heads, max_tokens, dtype=factor_dtype, **z)   # float32 or float16
        self.c_k = torch.zeros(batch, n_kv_heads, head_dim, dtype=torch.float32, **z)
        self.c_q = torch.zeros(batch, n_q_heads, head_dim, dtype=torch.float32, **z) if with_cq else None
        self.f_bias = torch.zeros(batch, n_q_heads, max_tokens, dtype=torch.float32, **z) if with_cq else None
        self.n_indexed = torch.zeros(batch, dtype=torch.int32, **z)
        self.n_total = torch.zeros(batch, dtype=torch.int32, **z)
        self.kv = rbq_kv(self.K.data_ptr(), self.V.data_ptr(), self.K.stride(0), self.K.stride(1), self.K.stride(2))
        self.idx = rbq_index(self.codes.data_ptr(), self.f_scale.data_ptr(),
                             None if self.f_bias is None else self.f_bias.data_ptr(), self.c_k.data_ptr(),
                             None if self.c_q is None else self.c_q.data_ptr(), self.n_indexed.data_ptr(),
                             self.n_total.data_ptr())

    def close(self):
        if self.ctx is not None:
            rbq_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # allocation helpers for outputs
    def new_scores(self):
        return torch.empty(self.B, self.Hq, self.Lcap, dtype=torch.float32, device=self.dev)

    def new_sel(self):
        return (torch.empty(self.B, self.Hq, self.Lcap, dtype=torch.int32, device=self.dev),
                torch.empty(self.B, self.Hq, dtype=torch.int32, device=self.dev))

    def new_out(self):
        return torch.empty(self.B, self.Hq, self.D, dtype=self.out_dtype, device=self.dev)

    # the calls
    def encode_keys(self, seq_lens: torch.Tensor, flags=0, stream=None):
        rbq_encode_keys(self.ctx, self.kv, seq_lens, flags, self.idx, stream)

    def append_tokens(self, k_new, v_new, stream=None, side_stream=None):
        rbq_append_tokens(self.ctx, k_new, v_new, k_new.shape[2], self.kv, self.idx, stream, side_stream)

    def query_quantize(self, q, qu=None, qparams=None, stream=None):
        rbq_query_quantize(self.ctx, q, self.idx, qu, qparams, stream)

    def int4_dot_binary(self, q, dot, pop, stream=None):
        rbq_int4_dot_binary(self.ctx, q, self.idx, dot, pop, stream)

    def estimate_scores(self, q, scores, stream=None):
        rbq_estimate_scores(self.ctx, q, self.idx, scores, stream)

    def topp_select(self, scores, p, sel_idx, sel_cnt, stream=None):
        rbq_topp_select(self.ctx, scores, self.idx, p, sel_idx, sel_cnt, stream)

    def topp_select_static(self, scores, p, sel_idx, sel_cnt, stream=None):
        rbq_topp_select_static(self.ctx, scores, self.idx, p, sel_idx, sel_cnt, stream)

    def topp_select_alg3(self, scores, p, sel_idx, sel_cnt, iters=None, stream=None):
        rbq_topp_select_alg3(self.ctx, scores, self.idx, p, sel_idx, sel_cnt, iters, stream)

    def sparse_attention(self, q, sel_idx, sel_cnt, out, lse=None, stream=None):
        rbq_sparse_attention(self.ctx, q, self.kv, self.idx, sel_idx, sel_cnt, out, lse, stream)

    def decode_step(self, q, p, out, sel_idx=None, sel_cnt=None, stream=None):
        rbq_decode_step(self.ctx, q, self.kv, self.idx, p, out, sel_idx, sel_cnt, stream)

    def decode_step_host(self, q_host, p, out_host, stream=None):
        rbq_decode_step_host(self.ctx, q_host, self.kv, self.idx, p, out_host, stream)

    def launch_count(self):
        return rbq_launch_count(self.ctx)

    def status_flags(self, stream=None):
        return rbq_status_flags(self.ctx, stream)

    def profile_enable(self, on=True):
        rbq_profile_enable(self.ctx, on)

    def profile_read(self):
        return rbq_profile_read(self.ctx)
