"""oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around ``m2r2_oracle.c`` (plain fp32 CPU implementation of the M2R2 hot path,
written from /root/reference/PAPER.md and DESIGN.md's readings).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It never imports ``paper_2502_02040_b200`` and shares no code with it;
inputs come from ``m2r2_synth`` (seeded generators, no method arithmetic).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "m2r2_oracle.c")
_LIB = os.path.join(_HERE, "libm2r2_oracle.so")

MAX_HEADS, MAX_GATES, MAX_LAYERS = 128, 16, 128

_TENSORS = ["embed", "gf", "lm_head", "lm_A", "lm_B",
            "g1", "g2", "wq", "wk", "wv", "wo", "wgate", "wup", "wdown",
            "Aq", "Bq", "Ak", "Bk", "Av", "Bv", "Ao", "Bo", "Ag", "Bg", "Au", "Bu", "Ad", "Bd",
            "router", "Ug", "Uu", "Ud", "ewg", "ewu", "ewd", "arla"]
_TID = {k: i for i, k in enumerate(_TENSORS)}


class _Config(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("n_layers", "d_model", "n_heads", "head_dim", "d_ff", "vocab", "dtype", "max_seq")] + \
               [("rms_eps", ctypes.c_float), ("rope_theta", ctypes.c_float),
                ("accel_enabled", ctypes.c_int32), ("n_accel_heads", ctypes.c_int32),
                ("accel_heads", ctypes.c_int32 * MAX_HEADS),
                ("adapter_rank", ctypes.c_int32), ("n_gates", ctypes.c_int32),
                ("gates", ctypes.c_int32 * MAX_GATES),
                ("accel_end_layer", ctypes.c_int32), ("lm_head_adapter", ctypes.c_int32),
                ("n_experts", ctypes.c_int32), ("top_k", ctypes.c_int32),
                ("d_ff_expert", ctypes.c_int32), ("cache_slots", ctypes.c_int32),
                ("accel_mlp_rank", ctypes.c_int32), ("renorm_topk", ctypes.c_int32),
                ("aot_lo", ctypes.c_int32 * MAX_LAYERS), ("aot_hi", ctypes.c_int32 * MAX_LAYERS),
                ("accel_topk_tokens", ctypes.c_int32), ("arla_dim", ctypes.c_int32)]


class _Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in
                ("steps", "drafted", "accepted", "emitted",
                 "expert_hits", "expert_misses", "prefetched", "on_demand")]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i32, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_float
        L.orc_create.restype = vp
        L.orc_create.argtypes = [ctypes.POINTER(_Config)]
        L.orc_destroy.argtypes = [vp]
        L.orc_reset.argtypes = [vp]
        L.orc_set_tensor.argtypes = [vp, i32, i32, i32, vp]
        L.orc_set_logit_script.argtypes = [vp, vp, vp, i32, i32, f32]
        L.orc_set_router_script.argtypes = [vp, vp, vp, i32, i32, f32]
        L.orc_set_policy.argtypes = [vp, i32]
        L.orc_prefill.argtypes = [vp, vp, i32, vp]
        L.orc_decode_step.argtypes = [vp, i32, vp, vp]
        L.orc_spec_step.argtypes = [vp, i32, vp, vp, vp]
        for name in ("orc_trace_h", "orc_trace_p", "orc_logits", "orc_route_idx", "orc_route_w",
                     "orc_pred_idx", "orc_lru"):
            getattr(L, name).restype = vp
            getattr(L, name).argtypes = [vp]
        for name in ("orc_exit_logits", "orc_kcache", "orc_vcache"):
            getattr(L, name).restype = vp
            getattr(L, name).argtypes = [vp, i32]
        L.orc_kv_len.argtypes = [vp]
        L.orc_pending.argtypes = [vp]
        L.orc_last_margin.restype = f32
        L.orc_last_margin.argtypes = [vp]
        L.orc_last_draft_margin.restype = f32
        L.orc_last_draft_margin.argtypes = [vp]
        L.orc_step_min_margin.restype = f32
        L.orc_step_min_margin.argtypes = [vp]
        L.orc_topk_margin.restype = f32
        L.orc_topk_margin.argtypes = [vp]
        L.orc_exit_score.restype = f32
        L.orc_exit_score.argtypes = [vp, ctypes.c_int32]
        L.orc_get_stats.argtypes = [vp, ctypes.POINTER(_Stats)]
        L.orc_rope.argtypes = [vp, vp, i32]
        L.orc_rmsnorm.argtypes = [vp, vp, vp, vp]
        L.orc_route.argtypes = [vp, vp, vp, vp, vp]
        L.orc_argmax.argtypes = [vp, i32]
        L.orc_accel_layer.argtypes = [vp, i32, vp, i32]
        L.orc_slow_layer.argtypes = [vp, i32, vp, i32, i32]
        L.orc_lru_use.argtypes = [vp, i32, vp]
        L.orc_lru_predict.argtypes = [vp, i32, vp]
        _lib = L
    return _lib


def _fill_config(c) -> _Config:
    s = _Config()
    for n in ("n_layers", "d_model", "n_heads", "head_dim", "d_ff", "vocab", "dtype", "max_seq",
              "adapter_rank", "accel_end_layer", "n_experts", "top_k", "d_ff_expert",
              "cache_slots", "accel_mlp_rank"):
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
    s.renorm_topk = int(c.renorm_topk)
    for i, (lo, hi) in enumerate(c.aot_targets):
        s.aot_lo[i], s.aot_hi[i] = lo, hi
    s.accel_topk_tokens = int(getattr(c, "accel_topk_tokens", 0))
    s.arla_dim = int(getattr(c, "arla_dim", 0))
    return s


class Oracle:
    """One sequence of the M2R2 decode path on the CPU.  `weights` is the dict produced by
    ``m2r2_synth.gen_weights`` (numpy arrays in storage dtype); the arrays are borrowed."""

    def __init__(self, cfg, weights):
        self.cfg = cfg
        self.W = weights  # keep alive
        self.L = lib()
        self._c = _fill_config(cfg)
        self.h = self.L.orc_create(ctypes.byref(self._c))
        for k in ("embed", "gf", "lm_head", "lm_A", "lm_B", "arla"):
            if k in weights:
                self._set(k, -1, 0, weights[k])
        for l, Lw in enumerate(weights["layers"]):
            for k, a in Lw.items():
                if k == "experts":
                    for e, E in enumerate(a):
                        for kk, aa in E.items():
                            self._set(kk, l, e, aa)
                else:
                    self._set(k, l, 0, a)

    def _set(self, kind, layer, expert, arr):
        assert arr.flags.c_contiguous
        assert arr.dtype == (np.float32 if self.cfg.dtype == 0 else np.uint16), (kind, arr.dtype)
        rc = self.L.orc_set_tensor(self.h, _TID[kind], layer, expert, arr.ctypes.data)
        assert rc == 0, (kind, layer, expert)

    def close(self):
        if self.h:
            self.L.orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- calls mirroring the C-ABI of the product ----
    def reset(self):
        self.L.orc_reset(self.h)

    def set_logit_script(self, full_tok, draft_tok, first_pos, beta=1000.0):
        if full_tok is None:
            self.L.orc_set_logit_script(self.h, None, None, 0, 0, 0.0)
            return
        f = np.ascontiguousarray(full_tok, dtype=np.int32)
        g = np.ascontiguousarray(draft_tok, dtype=np.int32)
        self.L.orc_set_logit_script(self.h, f.ctypes.data, g.ctypes.data, first_pos, len(f), beta)

    def set_router_script(self, actual, pred, first_pos, beta=1000.0):
        if actual is None:
            self.L.orc_set_router_script(self.h, None, None, 0, 0, 0.0)
            return
        a = np.ascontiguousarray(actual, dtype=np.int32)
        p = np.ascontiguousarray(pred, dtype=np.int32)
        self.L.orc_set_router_script(self.h, a.ctypes.data, p.ctypes.data, first_pos, a.shape[0], beta)

    def set_policy(self, policy):
        assert self.L.orc_set_policy(self.h, policy) == 0

    def prefill(self, tokens) -> int:
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        out = ctypes.c_int32(0)
        rc = self.L.orc_prefill(self.h, t.ctypes.data, len(t), ctypes.byref(out))
        assert rc == 0, rc
        return out.value

    def decode_step(self, force_token=None):
        """-> (token, exit_tokens[J])"""
        out = ctypes.c_int32(0)
        ex = np.full(max(1, len(self.cfg.gates)), -1, dtype=np.int32)
        rc = self.L.orc_decode_step(self.h, -1 if force_token is None else int(force_token),
                                    ctypes.byref(out), ex.ctypes.data)
        assert rc == 0, rc
        return out.value, ex[:len(self.cfg.gates)].copy()

    def spec_step(self, gamma):
        """-> (accepted tokens list, drafts list)"""
        acc = np.zeros(gamma + 1, dtype=np.int32)
        dr = np.zeros(max(1, gamma), dtype=np.int32)
        n = ctypes.c_int32(0)
        rc = self.L.orc_spec_step(self.h, gamma, acc.ctypes.data, ctypes.byref(n), dr.ctypes.data)
        assert rc == 0, rc
        return acc[:n.value].tolist(), dr[:gamma].tolist()

    # ---- introspection ----
    def _view(self, ptr, shape, dtype=np.float32):
        n = int(np.prod(shape))
        ct = {np.float32: ctypes.c_float, np.int32: ctypes.c_int32}[dtype]
        buf = (ct * n).from_address(ptr)
        return np.frombuffer(buf, dtype=dtype).reshape(shape)

    @property
    def kv_len(self):
        return self.L.orc_kv_len(self.h)

    @property
    def pending(self):
        return self.L.orc_pending(self.h)

    def trace_h(self):
        return self._view(self.L.orc_trace_h(self.h), (self.cfg.n_layers + 1, self.cfg.d_model)).copy()

    def trace_p(self):
        return self._view(self.L.orc_trace_p(self.h), (self.cfg.n_layers + 1, self.cfg.d_model)).copy()

    def logits(self):
        return self._view(self.L.orc_logits(self.h), (self.cfg.vocab,)).copy()

    def exit_logits(self, gate):
        return self._view(self.L.orc_exit_logits(self.h, gate), (self.cfg.vocab,)).copy()

    def margin(self):
        return float(self.L.orc_last_margin(self.h))

    def draft_margin(self):
        return float(self.L.orc_last_draft_margin(self.h))

    def exit_scores(self):
        """ARLA exit score of every gate for the last decode_step"""
        return np.array([self.L.orc_exit_score(self.h, j) for j in range(len(self.cfg.gates))], dtype=np.float32)

    def topk_margin(self):
        """smallest gap between the k-th and (k+1)-th slow attention score of any top-k token selection of the last step"""
        return float(self.L.orc_topk_margin(self.h))

    def step_margin(self):
        """smallest top-2 margin of any argmax (every draft, every verify row) of the last step"""
        return float(self.L.orc_step_min_margin(self.h))

    def kcache(self, layer):
        """writable view [max_seq, d] (tests poison dead positions through it)"""
        return self._view(self.L.orc_kcache(self.h, layer), (self.cfg.max_seq, self.cfg.d_model))

    def vcache(self, layer):
        return self._view(self.L.orc_vcache(self.h, layer), (self.cfg.max_seq, self.cfg.d_model))

    def route_idx(self):
        return self._view(self.L.orc_route_idx(self.h), (self.cfg.n_layers, self.cfg.top_k), np.int32).copy()

    def route_w(self):
        return self._view(self.L.orc_route_w(self.h), (self.cfg.n_layers, self.cfg.top_k)).copy()

    def pred_idx(self):
        return self._view(self.L.orc_pred_idx(self.h), (self.cfg.n_layers, self.cfg.top_k), np.int32).copy()

    def lru(self):
        return self._view(self.L.orc_lru(self.h), (self.cfg.n_layers, self.cfg.cache_slots), np.int32).copy()

    def stats(self) -> dict:
        s = _Stats()
        self.L.orc_get_stats(self.h, ctypes.byref(s))
        return {n: getattr(s, n) for n, _ in _Stats._fields_}

    # ---- stand-alone pieces for the pins ----
    def rope(self, v, t):
        v = np.ascontiguousarray(v, dtype=np.float32).copy()
        self.L.orc_rope(self.h, v.ctypes.data, t)
        return v

    def route(self, Wr, y):
        idx = np.zeros(self.cfg.top_k, dtype=np.int32)
        w = np.zeros(self.cfg.top_k, dtype=np.float32)
        y = np.ascontiguousarray(y, dtype=np.float32)
        self.L.orc_route(self.h, Wr.ctypes.data, y.ctypes.data, idx.ctypes.data, w.ctypes.data)
        return idx, w

    def argmax(self, v):
        v = np.ascontiguousarray(v, dtype=np.float32)
        return self.L.orc_argmax(v.ctypes.data, len(v))

    def accel_layer(self, i, p, t):
        p = np.ascontiguousarray(p, dtype=np.float32).copy()
        self.L.orc_accel_layer(self.h, i, p.ctypes.data, t)
        return p

    def slow_layer(self, i, h, t0):
        h = np.ascontiguousarray(h, dtype=np.float32).copy()
        m = 1 if h.ndim == 1 else h.shape[0]
        self.L.orc_slow_layer(self.h, i, h.ctypes.data, m, t0)
        return h

    def lru_use(self, L, idx):
        a = np.ascontiguousarray(idx, dtype=np.int32)
        self.L.orc_lru_use(self.h, L, a.ctypes.data)

    def lru_predict(self, L, idx):
        a = np.ascontiguousarray(idx, dtype=np.int32)
        self.L.orc_lru_predict(self.h, L, a.ctypes.data)
