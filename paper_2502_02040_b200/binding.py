"""Thin ctypes binding of include/m2r2.h — argument marshalling only.

Every step of the path runs in the CUDA kernels of libm2r2.so; torch is used for device
memory, pinned host memory and streams.  There is NO CPU fallback: importing this module
without the built library raises, and every call needs a CUDA device.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from . import build as _build

MAX_HEADS, MAX_GATES, MAX_LAYERS, MAX_BATCH, MAX_DRAFT = 128, 16, 128, 8, 7
OK, INVALID_ARG, BAD_STATE, CAPACITY, CUDA, UNSUPPORTED = 0, -1, -2, -3, -4, -5
FP32, BF16 = 0, 1
POLICY_FIXED, POLICY_LRU, POLICY_LRU_AOT, POLICY_LRU_RANDOM, POLICY_LRU_PREV = 0, 1, 2, 3, 4
DBG_H, DBG_P, DBG_LOGITS, DBG_EXIT_LOGITS, DBG_K, DBG_V, DBG_ROUTE_IDX, DBG_ROUTE_W, DBG_PRED_IDX, DBG_EXIT_SCORE = range(10)

i32, i64, u32, u64, f32, vp = (ctypes.c_int32, ctypes.c_int64, ctypes.c_uint32, ctypes.c_uint64,
                               ctypes.c_float, ctypes.c_void_p)


class Config(ctypes.Structure):
    _fields_ = [("struct_size", u32)] + \
               [(n, i32) for n in ("n_layers", "d_model", "n_heads", "head_dim", "d_ff", "vocab",
                                   "dtype", "max_batch", "max_seq")] + \
               [("rms_eps", f32), ("rope_theta", f32),
                ("accel_enabled", i32), ("n_accel_heads", i32), ("accel_heads", i32 * MAX_HEADS),
                ("adapter_rank", i32), ("n_gates", i32), ("gates", i32 * MAX_GATES),
                ("accel_end_layer", i32), ("lm_head_adapter", i32), ("exit_heads_enabled", i32),
                ("n_experts", i32), ("top_k", i32), ("d_ff_expert", i32),
                ("cache_slots_per_layer", i32), ("accel_mlp_rank", i32), ("renorm_topk", i32),
                ("aot_lo", i32 * MAX_LAYERS), ("aot_hi", i32 * MAX_LAYERS), ("accel_topk_tokens", i32), ("arla_dim", i32)]


class Sizes(ctypes.Structure):
    _fields_ = [(n, u64) for n in ("weights_bytes", "kv_bytes", "scratch_bytes",
                                   "expert_cache_bytes", "expert_store_bytes")]


class Buffers(ctypes.Structure):
    _fields_ = [(n, vp) for n in ("weights", "kv", "scratch", "expert_cache")]


_LAYER_FIELDS = ["g1", "g2", "wq", "wk", "wv", "wo", "wgate", "wup", "wdown",
                 "Aq", "Bq", "Ak", "Bk", "Av", "Bv", "Ao", "Bo", "Ag", "Bg", "Au", "Bu", "Ad", "Bd",
                 "router", "Ug", "Uu", "Ud"]


class LayerWeights(ctypes.Structure):
    _fields_ = [(n, vp) for n in _LAYER_FIELDS] + \
               [("expert_gate", ctypes.POINTER(vp)), ("expert_up", ctypes.POINTER(vp)),
                ("expert_down", ctypes.POINTER(vp))]


class WeightTable(ctypes.Structure):
    _fields_ = [("embed", vp), ("gf", vp), ("lm_head", vp), ("lm_A", vp), ("lm_B", vp),
                ("layers", ctypes.POINTER(LayerWeights)), ("arla", vp)]


class Stats(ctypes.Structure):
    _fields_ = [("kv_len", i32 * MAX_BATCH)] + \
               [(n, i64) for n in ("steps", "drafted", "accepted", "emitted", "expert_hits",
                                   "expert_misses", "expert_prefetched", "expert_on_demand",
                                   "h2d_bytes", "algorithmic_bytes_last", "kernel_launches")]


PROF_CLASSES = ["qkv", "rope_append", "attention", "o_proj", "gate_up", "down", "heads", "other", "fused_step", "_"]


class Profile(ctypes.Structure):
    _fields_ = [("ms", ctypes.c_double * 10), ("segments", i64 * 10), ("steps", i64)]


EXPORTS = ["m2r2_query_sizes", "m2r2_create", "m2r2_destroy", "m2r2_load_weights", "m2r2_prefill",
           "m2r2_decode_step", "m2r2_spec_step", "m2r2_moe_prefetch", "m2r2_set_policy",
           "m2r2_set_logit_script", "m2r2_set_router_script", "m2r2_get_stats", "m2r2_debug_read",
           "m2r2_reset", "m2r2_set_fused", "m2r2_set_profile", "m2r2_get_profile", "m2r2_last_error",
           "m2r2_version", "m2r2_final_head_noalloc", "m2r2_noalloc_last_error"]

_lib = None


_lib_path = None   # tests may point the binding at a variant build of the library (use_library)


def use_library(path):
    """Load `path` instead of the in-tree libm2r2.so from now on (None: back to the default).  Test hook for variant
    builds (build.build_variant); engines created earlier keep the library they were created with."""
    global _lib, _lib_path
    _lib, _lib_path = None, path


def lib():
    """Load libm2r2.so (building it with nvcc if the in-tree copy is missing or stale)."""
    global _lib
    if _lib is None:
        path = _lib_path or _build.build()
        L = ctypes.CDLL(path)
        L.m2r2_query_sizes.argtypes = [ctypes.POINTER(Config), ctypes.POINTER(Sizes)]
        L.m2r2_create.argtypes = [ctypes.POINTER(Config), ctypes.POINTER(Buffers), vp, vp, ctypes.POINTER(vp)]
        L.m2r2_destroy.argtypes = [vp]
        L.m2r2_load_weights.argtypes = [vp, ctypes.POINTER(WeightTable)]
        L.m2r2_prefill.argtypes = [vp, vp, i32, i32, vp]
        L.m2r2_decode_step.argtypes = [vp, vp, vp, vp]
        L.m2r2_spec_step.argtypes = [vp, i32, vp, vp]
        L.m2r2_moe_prefetch.argtypes = [vp, i32, vp, i32]
        L.m2r2_set_policy.argtypes = [vp, i32]
        L.m2r2_set_logit_script.argtypes = [vp, vp, vp, i32, i32, f32]
        L.m2r2_set_router_script.argtypes = [vp, vp, vp, i32, i32, f32]
        L.m2r2_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
        L.m2r2_debug_read.argtypes = [vp, i32, i32, i32, vp, ctypes.c_size_t]
        L.m2r2_reset.argtypes = [vp]
        L.m2r2_set_fused.argtypes = [vp, i32]
        L.m2r2_set_profile.argtypes = [vp, i32]
        L.m2r2_get_profile.argtypes = [vp, ctypes.POINTER(Profile)]
        L.m2r2_last_error.argtypes = [vp]
        L.m2r2_last_error.restype = ctypes.c_char_p
        L.m2r2_version.restype = ctypes.c_char_p
        L.m2r2_final_head_noalloc.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, f32, vp]
        L.m2r2_noalloc_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def make_config(c) -> Config:
    """m2r2_synth.ModelConfig (or anything with the same attributes) -> m2r2_config."""
    s = Config()
    s.struct_size = ctypes.sizeof(Config)
    for n in ("n_layers", "d_model", "n_heads", "head_dim", "d_ff", "vocab", "dtype", "max_batch",
              "max_seq", "adapter_rank", "accel_end_layer", "n_experts", "top_k", "d_ff_expert",
              "accel_mlp_rank"):
        setattr(s, n, int(getattr(c, n)))
    s.rms_eps, s.rope_theta = c.rms_eps, c.rope_theta
    s.accel_enabled = int(c.accel_enabled)
    s.n_accel_heads = len(c.accel_heads)
    for i, a in enumerate(c.accel_heads):
        s.accel_heads[i] = a
    s.n_gates = len(c.gates)
    for i, g in enumerate(c.gates):
        s.gates[i] = g
    s.lm_head_adapter = int(c.lm_head_adapter)
    s.exit_heads_enabled = int(getattr(c, "exit_heads_enabled", True))
    s.cache_slots_per_layer = int(c.cache_slots)
    s.renorm_topk = int(c.renorm_topk)
    for i, (lo, hi) in enumerate(c.aot_targets):
        s.aot_lo[i], s.aot_hi[i] = lo, hi
    s.accel_topk_tokens = int(getattr(c, "accel_topk_tokens", 0))
    s.arla_dim = int(getattr(c, "arla_dim", 0))
    return s


class M2R2Error(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("m2r2 status %d: %s" % (code, msg))
        self.code = code


class Engine:
    """Owns the torch buffers and streams a context borrows, and exposes the C-ABI calls under
    their own names (prefill, decode_step, spec_step, moe_prefetch, ...)."""

    def __init__(self, cfg, weights: Optional[dict] = None, exit_heads: bool = True, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2502_02040_b200 needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.cfg = cfg
        self.L = lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.c = make_config(cfg)
        self.c.exit_heads_enabled = int(exit_heads)
        sz = Sizes()
        self._chk(self.L.m2r2_query_sizes(ctypes.byref(self.c), ctypes.byref(sz)), "query_sizes")
        self.sizes = sz
        alloc = lambda n: torch.empty(max(int(n), 256), dtype=torch.uint8, device=self.device)
        self.buf_w, self.buf_kv, self.buf_s = alloc(sz.weights_bytes), alloc(sz.kv_bytes), alloc(sz.scratch_bytes)
        self.buf_s.zero_()
        self.buf_kv.zero_()
        self.buf_e = alloc(sz.expert_cache_bytes) if sz.expert_cache_bytes else None
        self.compute_stream = torch.cuda.Stream(device=self.device)
        self.copy_stream = torch.cuda.Stream(device=self.device)
        torch.cuda.synchronize()
        bufs = Buffers(self.buf_w.data_ptr(), self.buf_kv.data_ptr(), self.buf_s.data_ptr(),
                       self.buf_e.data_ptr() if self.buf_e is not None else None)
        h = vp()
        rc = self.L.m2r2_create(ctypes.byref(self.c), ctypes.byref(bufs), vp(self.compute_stream.cuda_stream),
                                vp(self.copy_stream.cuda_stream), ctypes.byref(h))
        if rc != OK:
            raise M2R2Error(rc, "m2r2_create failed")
        self.h = h
        self._keep = []
        self.B = 0
        if weights is not None:
            self.load_weights(weights)

    # ------------------------------------------------------------------ helpers
    def _chk(self, rc, what=""):
        if rc < 0:
            msg = self.L.m2r2_last_error(self.h).decode() if getattr(self, "h", None) else what
            raise M2R2Error(rc, what + ": " + msg)
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.L.m2r2_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _ptr(a):
        return None if a is None else vp(a.ctypes.data)

    # ------------------------------------------------------------------ C-ABI calls
    def load_weights(self, W: dict):
        """W: dict from m2r2_synth.gen_weights (numpy arrays in storage dtype).  Expert blobs
        must already live in pinned host memory (use `pinned_expert_alloc`)."""
        cfg = self.cfg
        layers = (LayerWeights * cfg.n_layers)()
        keep = []
        for i, Lw in enumerate(W["layers"]):
            for n in _LAYER_FIELDS:
                if n in Lw:
                    a = Lw[n]
                    assert a.flags.c_contiguous
                    setattr(layers[i], n, a.ctypes.data)
            if cfg.n_experts:
                for field, key in (("expert_gate", "ewg"), ("expert_up", "ewu"), ("expert_down", "ewd")):
                    arr = (vp * cfg.n_experts)(*[E[key].ctypes.data for E in Lw["experts"]])
                    keep.append(arr)
                    setattr(layers[i], field, ctypes.cast(arr, ctypes.POINTER(vp)))
        t = WeightTable()
        for n in ("embed", "gf", "lm_head", "lm_A", "lm_B", "arla"):
            if n in W:
                setattr(t, n, W[n].ctypes.data)
        t.layers = ctypes.cast(layers, ctypes.POINTER(LayerWeights))
        self._keep = [W, keep, layers]   # expert blobs are read by DMA for the ctx lifetime
        self._chk(self.L.m2r2_load_weights(self.h, ctypes.byref(t)), "load_weights")

    def pinned_expert_alloc(self):
        """Allocator for m2r2_synth.gen_weights(expert_alloc=...): numpy views of pinned memory."""
        torch = self.torch
        np_dt = np.float32 if self.cfg.dtype == FP32 else np.uint16
        t_dt = torch.float32 if self.cfg.dtype == FP32 else torch.int16
        pool = []

        def alloc(shape):
            t = torch.empty(int(np.prod(shape)), dtype=t_dt).pin_memory()
            pool.append(t)
            return t.numpy().view(np_dt).reshape(shape)
        self._pinned_pool = pool
        return alloc

    def prefill(self, tokens):
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        if t.ndim == 1:
            t = t[None]
        B, P = t.shape
        out = np.zeros(B, dtype=np.int32)
        self._chk(self.L.m2r2_prefill(self.h, self._ptr(t), B, P, self._ptr(out)), "prefill")
        self.B = B
        return out

    def decode_step(self, force_tokens=None, want_tokens=True, want_exit=False):
        B = self.B
        f = None if force_tokens is None else np.ascontiguousarray(np.atleast_1d(force_tokens), dtype=np.int32)
        out = np.zeros(B, dtype=np.int32) if want_tokens else None
        ex = np.full((B, max(1, len(self.cfg.gates))), -1, dtype=np.int32) if want_exit else None
        self._chk(self.L.m2r2_decode_step(self.h, self._ptr(f), self._ptr(out), self._ptr(ex)), "decode_step")
        return (out, ex) if want_exit else out

    def spec_step(self, k):
        B = self.B
        acc = np.zeros((B, k + 1), dtype=np.int32)
        n = np.zeros(B, dtype=np.int32)
        self._chk(self.L.m2r2_spec_step(self.h, k, self._ptr(acc), self._ptr(n)), "spec_step")
        return acc, n

    def moe_prefetch(self, src_layer=0, pairs=None):
        if pairs is None:
            return self._chk(self.L.m2r2_moe_prefetch(self.h, src_layer, None, 0), "moe_prefetch")
        p = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        return self._chk(self.L.m2r2_moe_prefetch(self.h, src_layer, self._ptr(p), len(p)), "moe_prefetch")

    def set_policy(self, policy):
        self._chk(self.L.m2r2_set_policy(self.h, policy), "set_policy")

    def set_logit_script(self, full_tok, draft_tok, first_pos, beta=1000.0):
        if full_tok is None:
            self._chk(self.L.m2r2_set_logit_script(self.h, None, None, 0, 0, 0.0))
            return
        B = self.cfg.max_batch
        f = np.ascontiguousarray(full_tok, dtype=np.int32).reshape(B, -1)
        g = np.ascontiguousarray(draft_tok, dtype=np.int32).reshape(B, -1)
        self._chk(self.L.m2r2_set_logit_script(self.h, self._ptr(f), self._ptr(g), first_pos, f.shape[1], beta), "set_logit_script")

    def set_router_script(self, actual, pred, first_pos, beta=1000.0):
        if actual is None:
            self._chk(self.L.m2r2_set_router_script(self.h, None, None, 0, 0, 0.0))
            return
        a = np.ascontiguousarray(actual, dtype=np.int32)
        p = np.ascontiguousarray(pred, dtype=np.int32)
        self._chk(self.L.m2r2_set_router_script(self.h, self._ptr(a), self._ptr(p), first_pos, a.shape[0], beta), "set_router_script")

    def get_stats(self) -> dict:
        s = Stats()
        self._chk(self.L.m2r2_get_stats(self.h, ctypes.byref(s)), "get_stats")
        d = {n: getattr(s, n) for n, _ in Stats._fields_ if n != "kv_len"}
        d["kv_len"] = list(s.kv_len)[:max(1, self.B)]
        return d

    def debug_read(self, what, layer=0, b=0, n=None):
        cfg = self.cfg
        if n is None:
            n = {DBG_H: cfg.d_model, DBG_P: cfg.d_model, DBG_LOGITS: cfg.vocab, DBG_EXIT_LOGITS: cfg.vocab,
                 DBG_ROUTE_IDX: cfg.n_layers * max(1, cfg.top_k), DBG_ROUTE_W: cfg.n_layers * max(1, cfg.top_k),
                 DBG_PRED_IDX: cfg.n_layers * max(1, cfg.top_k), DBG_EXIT_SCORE: max(1, len(cfg.gates))}[what]
        out = np.zeros(n, dtype=np.float32)
        self._chk(self.L.m2r2_debug_read(self.h, what, layer, b, self._ptr(out), n), "debug_read")
        return out

    def kcache(self, layer, T, b=0, v=False):
        out = self.debug_read(DBG_V if v else DBG_K, layer, b, T * self.cfg.d_model)
        return out.reshape(T, self.cfg.d_model)

    def reset(self):
        self._chk(self.L.m2r2_reset(self.h), "reset")
        self.B = 0

    def set_fused(self, on: bool):
        self._chk(self.L.m2r2_set_fused(self.h, int(on)), "set_fused")

    def set_profile(self, on: bool):
        self._chk(self.L.m2r2_set_profile(self.h, int(on)), "set_profile")

    def get_profile(self) -> dict:
        """-> {"steps": n, "ms": {class: ms per step}, "segments": {class: segments per step}}"""
        p = Profile()
        self._chk(self.L.m2r2_get_profile(self.h, ctypes.byref(p)), "get_profile")
        n = max(1, p.steps)
        return {"steps": p.steps,
                "ms": {c: p.ms[i] / n for i, c in enumerate(PROF_CLASSES) if p.segments[i]},
                "segments": {c: p.segments[i] / n for i, c in enumerate(PROF_CLASSES) if p.segments[i]}}

    def sync(self):
        self.compute_stream.synchronize()


# ------------------------------------------------------------------ the entry point that allocates nothing
NOALLOC_MAX_ROWS, NOALLOC_MAX_D = 8, 8192


def final_head_noalloc(h, g_f, w_lm, logits, dtype, rms_eps, stream=None):
    """m2r2_final_head_noalloc (include/m2r2.h): logits[row] = W_lm . rms(h[row]; g_f) with the op's scratch in a static
    device array of the library — no allocation in the call.  All arguments are CUDA torch tensors on the current device:
    h fp32 [m][d] contiguous, g_f [d] and w_lm [vocab][d] in the storage dtype (fp32, or bf16 / its int16 bit pattern),
    logits fp32 [m][vocab] (written).  `stream`: a torch.cuda.Stream or None (torch's current stream).  Calls that
    overlap on the GPU race on the shared scratch."""
    import torch
    assert h.is_cuda and g_f.is_cuda and w_lm.is_cuda and logits.is_cuda
    assert h.dtype == torch.float32 and logits.dtype == torch.float32
    assert h.is_contiguous() and g_f.is_contiguous() and w_lm.is_contiguous() and logits.is_contiguous()
    m, d = h.shape
    vocab = w_lm.shape[0]
    assert tuple(w_lm.shape) == (vocab, d) and g_f.numel() == d and tuple(logits.shape) == (m, vocab)
    st = stream if stream is not None else torch.cuda.current_stream(h.device)
    L = lib()
    rc = L.m2r2_final_head_noalloc(vp(h.data_ptr()), vp(g_f.data_ptr()), vp(w_lm.data_ptr()), vp(logits.data_ptr()),
                                   int(m), int(d), int(vocab), int(dtype), float(rms_eps), vp(st.cuda_stream))
    if rc != OK:
        raise M2R2Error(rc, L.m2r2_noalloc_last_error().decode())
    return logits
