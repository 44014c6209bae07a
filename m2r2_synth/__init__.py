"""m2r2_synth — seeded synthetic inputs shared by the oracle and the CUDA path.

Holds the *input recipe* only (DESIGN.md §"Input recipe"): model-shape
configs taken from BASELINE.json, the counter-based PRNG (``synth.c``), random-init
weights N(0, 0.02) rounded to the storage dtype, uniform-random prompts, and the two
integer "scripts" (forced acceptance / seeded routing).  None of the method's arithmetic
lives here, and this module imports neither ``oracle`` nor ``paper_2502_02040_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field, replace
from typing import Callable, Dict, List, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth.c")
_LIB = os.path.join(_HERE, "libm2r2_synth.so")

FP32 = 0
BF16 = 1


def build(force: bool = False) -> str:
    """Compile synth.c with gcc (in-tree, next to the source)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, i32, f32, f64, vp = (ctypes.c_uint64, ctypes.c_int32, ctypes.c_float,
                                  ctypes.c_double, ctypes.c_void_p)
        lib.synth_normal_f32.argtypes = [u64, u64, u64, u64, f32, f32, vp]
        lib.synth_normal_bf16.argtypes = [u64, u64, u64, u64, f32, f32, vp]
        lib.synth_tokens.argtypes = [u64, u64, u64, i32, vp]
        lib.synth_logit_script.argtypes = [u64, u64, u64, i32, f64, vp, vp]
        lib.synth_router_script.argtypes = [u64, u64, i32, i32, i32, f64, f64, vp, vp]
        for f in (lib.synth_normal_f32, lib.synth_normal_bf16, lib.synth_tokens,
                  lib.synth_logit_script, lib.synth_router_script):
            f.restype = None
        _lib = lib
    return _lib


# --------------------------------------------------------------------------------------
# Model-shape configs (BASELINE.json `configs`; SURVEY.md §8 "Config shorthand")
# --------------------------------------------------------------------------------------
@dataclass(frozen=True)
class ModelConfig:
    name: str
    n_layers: int
    d_model: int
    n_heads: int
    head_dim: int
    d_ff: int
    vocab: int
    dtype: int = BF16              # storage dtype of weights and KV cache
    max_batch: int = 1
    max_seq: int = 1024
    rms_eps: float = 1e-5
    rope_theta: float = 10000.0
    # accelerated stream (§2.2, §2.5)
    accel_enabled: bool = True
    accel_heads: Tuple[int, ...] = ()
    adapter_rank: int = 8          # rank 8
    gates: Tuple[int, ...] = ()    # exit layers E_1 < ... < E_J
    accel_end_layer: int = 0       # accelerated stream runs in layers [0, accel_end_layer)
    lm_head_adapter: bool = False  # PAPER.md L162 "low-rank layers for ... language modeling heads"
    # MoE (§2.3.3)
    n_experts: int = 0
    top_k: int = 0
    d_ff_expert: int = 0
    cache_slots: int = 0
    accel_mlp_rank: int = 0
    renorm_topk: bool = True
    aot_targets: Tuple[Tuple[int, int], ...] = ()   # per source layer: [lo, hi) target layers
    accel_topk_tokens: int = 0                      # p attends the slow stream's top-k cached positions (0 = all)
    arla_dim: int = 0                               # latent dimension d^s of the exit router (0 = no ARLA)
    seed: int = 0x4D325232

    @property
    def is_moe(self) -> bool:
        return self.n_experts > 0

    @property
    def n_accel_heads(self) -> int:
        return len(self.accel_heads)

    @property
    def elt_bytes(self) -> int:
        return 4 if self.dtype == FP32 else 2


def aot_targets_for_rate(n_layers: int, rate: int, n_sources: Optional[int] = None):
    """PAPER.md L137/L244/L387: with a `rate`x stream, source layer i targets
    {rate*(i+1), ..., rate*(i+1)+rate-1} clipped to [0, N).  rate=2 -> {2i+2, 2i+3}."""
    out = []
    for i in range(n_layers):
        lo = min(rate * (i + 1), n_layers)
        hi = min(rate * (i + 1) + rate, n_layers)
        if n_sources is not None and i >= n_sources:
            lo = hi = 0
        out.append((lo, hi) if lo < hi else (0, 0))
    return tuple(out)


def config_c1() -> ModelConfig:
    """BASELINE.json configs[0]: tiny fp32 decoder; accel heads 2 of 8; gate at layer 2."""
    return ModelConfig(name="C1-tiny-fp32", n_layers=4, d_model=256, n_heads=8, head_dim=32,
                       d_ff=1024, vocab=2048, dtype=FP32, max_seq=128,
                       accel_heads=(0, 1), gates=(2,), accel_end_layer=2,
                       seed=0x4D325232 + 1)


def config_c2() -> ModelConfig:
    """BASELINE.json configs[1]: 3.8B-class bf16, both streams in every layer
    (gates {8,16,24}, accel in all 32 layers)."""
    return ModelConfig(name="C2-3.8B-bf16", n_layers=32, d_model=3072, n_heads=32, head_dim=96,
                       d_ff=8192, vocab=32064, dtype=BF16, max_seq=1024,
                       accel_heads=tuple(range(8)), gates=(8, 16, 24), accel_end_layer=32,
                       seed=0x4D325232 + 2)


def config_c3() -> ModelConfig:
    """BASELINE.json configs[2]: same model, self-spec from the layer-8 accelerated stream."""
    return replace(config_c2(), name="C3-3.8B-selfspec", gates=(8,), accel_end_layer=8,
                   lm_head_adapter=True)


def config_c4() -> ModelConfig:
    """BASELINE.json configs[3]: batch 8 x 4096-token KV, self-spec k=4."""
    return replace(config_c3(), name="C4-3.8B-b8-kv4096", max_batch=8, max_seq=4096 + 768)


def config_c5() -> ModelConfig:
    """BASELINE.json configs[4]: MoE bf16, 8 experts top-2, cache 2 experts/layer,
    prediction from the layer-4 accelerated residual (literal reading)."""
    n = 16
    tg = [(0, 0)] * n
    tg[3] = (4, n)          # p leaving layer 3 (= "layer-4 accelerated residual") targets layers 4..15
    return ModelConfig(name="C5-moe-bf16", n_layers=n, d_model=2048, n_heads=16, head_dim=128,
                       d_ff=0, vocab=32064, dtype=BF16, max_seq=768,
                       accel_heads=(0, 1, 2, 3), gates=(4,), accel_end_layer=4,
                       n_experts=8, top_k=2, d_ff_expert=5632, cache_slots=2, accel_mlp_rank=64,
                       aot_targets=tuple(tg), seed=0x4D325232 + 5)


def config_gemma7b_class() -> ModelConfig:
    """the regime of the paper's 2.8x (footnote 3 L133: Gemma-7B, drafts from the
    first 4 layers' accelerated stream, draft length 3): a 7B-class decoder whose 256k-row LM head dominates a draft.
    28 layers, d 3072, FFN 16384, vocab 256000, E = 4; 24 heads x 128 instead of Gemma's 16 x 256 and FFN 16384 instead
    of 24576 (the fused kernel's limits: d_h <= 128, F <= 16384) -- 6.9 B parameters."""
    return ModelConfig(name="Gemma7B-class-bf16", n_layers=28, d_model=3072, n_heads=24, head_dim=128,
                       d_ff=16384, vocab=256000, dtype=BF16, max_seq=1024,
                       accel_heads=tuple(range(6)), gates=(4,), accel_end_layer=4, lm_head_adapter=True,
                       seed=0x4D325232 + 7)


def config_olmoe_shaped() -> ModelConfig:
    """an OLMoE-shaped MoE decoder for the paper's five expert-loading strategies:
    16 layers, d 2048, 16 x 128 heads, 64 experts of FFN 1024 per layer, top-8, HALF of the experts resident (32 slots
    per layer), accelerated stream in layers 0..7 predicting with the paper's 2x schedule (layer i -> {2i+2, 2i+3})."""
    n = 16
    return ModelConfig(name="OLMoE-shaped-bf16", n_layers=n, d_model=2048, n_heads=16, head_dim=128,
                       d_ff=0, vocab=32064, dtype=BF16, max_seq=768,
                       accel_heads=(0, 1, 2, 3), gates=(8,), accel_end_layer=8,
                       n_experts=64, top_k=8, d_ff_expert=1024, cache_slots=32, accel_mlp_rank=64,
                       aot_targets=aot_targets_for_rate(n, 2, 8), seed=0x4D325232 + 6)


def config_small_bf16(**kw) -> ModelConfig:
    """Reduced bf16 dense model for parity tests: same structure as C2/C3 (head_dim 96,
    ragged row counts), sized so the oracle finishes in seconds."""
    base = ModelConfig(name="S-bf16", n_layers=6, d_model=384, n_heads=4, head_dim=96,
                       d_ff=1000, vocab=3001, dtype=BF16, max_seq=256,
                       accel_heads=(0, 2), gates=(2, 4), accel_end_layer=6,
                       seed=0x4D325232 + 11)
    return replace(base, **kw)


def config_small_moe(**kw) -> ModelConfig:
    """Reduced MoE model for parity tests (structure of C5)."""
    n = 6
    base = ModelConfig(name="S-moe", n_layers=n, d_model=256, n_heads=4, head_dim=64, d_ff=0,
                       vocab=1500, dtype=BF16, max_seq=256, accel_heads=(1, 3), gates=(),
                       accel_end_layer=n, n_experts=8, top_k=2, d_ff_expert=320, cache_slots=2,
                       accel_mlp_rank=16, aot_targets=aot_targets_for_rate(n, 2),
                       seed=0x4D325232 + 12)
    return replace(base, **kw)


# --------------------------------------------------------------------------------------
# Tensor inventory
# --------------------------------------------------------------------------------------
# kind ids (stable: they feed the PRNG key)
_KINDS = ["embed", "gf", "lm_head", "lm_A", "lm_B",
          "g1", "g2", "wq", "wk", "wv", "wo", "wgate", "wup", "wdown",
          "Aq", "Bq", "Ak", "Bk", "Av", "Bv", "Ao", "Bo", "Ag", "Bg", "Au", "Bu", "Ad", "Bd",
          "router", "Ug", "Uu", "Ud", "ewg", "ewu", "ewd", "arla"]
KIND_ID = {k: i for i, k in enumerate(_KINDS)}
GLOBAL_KINDS = ("embed", "gf", "lm_head", "lm_A", "lm_B", "arla")
EXPERT_KINDS = ("ewg", "ewu", "ewd")


def tensor_id(kind: str, layer: int = -1, expert: int = 0) -> int:
    return KIND_ID[kind] + 64 * (layer + 1) + 64 * 256 * expert


def global_shapes(c: ModelConfig) -> Dict[str, Tuple[int, ...]]:
    s = {"embed": (c.vocab, c.d_model), "gf": (c.d_model,), "lm_head": (c.vocab, c.d_model)}
    if c.lm_head_adapter:
        s["lm_A"] = (c.adapter_rank, c.d_model)
        s["lm_B"] = (c.vocab, c.adapter_rank)
    if c.arla_dim and c.accel_enabled and len(c.gates):
        # ARLA exit router, one block per gate: W_q^s, W_k^s, W_v^s [d^s, d] each, then one row holding w_o[0..d^s) and b
        s["arla"] = (len(c.gates) * (3 * c.arla_dim + 1), c.d_model)
    return s


def layer_shapes(c: ModelConfig, layer: int) -> Dict[str, Tuple[int, ...]]:
    """Row-major [out, in] shapes of one layer's tensors (SURVEY §8(b) load_weights)."""
    d, F, r = c.d_model, c.d_ff, c.adapter_rank
    da = c.n_accel_heads * c.head_dim
    s = {"g1": (d,), "g2": (d,), "wq": (d, d), "wk": (d, d), "wv": (d, d), "wo": (d, d)}
    accel = c.accel_enabled and layer < c.accel_end_layer
    if accel:
        s.update({"Aq": (r, d), "Bq": (da, r), "Ak": (r, d), "Bk": (da, r),
                  "Av": (r, d), "Bv": (da, r), "Ao": (r, da), "Bo": (d, r)})
    if c.is_moe:
        s["router"] = (c.n_experts, d)
        if accel:
            rm = c.accel_mlp_rank
            s.update({"Ug": (rm, d), "Uu": (rm, d), "Ud": (d, rm)})
    else:
        s.update({"wgate": (F, d), "wup": (F, d), "wdown": (d, F)})
        if accel:
            s.update({"Ag": (r, d), "Bg": (F, r), "Au": (r, d), "Bu": (F, r),
                      "Ad": (r, F), "Bd": (d, r)})
    return s


def expert_shapes(c: ModelConfig) -> Dict[str, Tuple[int, ...]]:
    return {"ewg": (c.d_ff_expert, c.d_model), "ewu": (c.d_ff_expert, c.d_model),
            "ewd": (c.d_model, c.d_ff_expert)}


def _np_dtype(c: ModelConfig):
    return np.float32 if c.dtype == FP32 else np.uint16


def gen_tensor(c: ModelConfig, kind: str, shape, layer: int = -1, expert: int = 0,
               out: Optional[np.ndarray] = None) -> np.ndarray:
    """One tensor: 0.02*normal (gains: 1 + 0.02*normal), storage dtype of `c`."""
    lib = _load()
    n = int(np.prod(shape))
    if out is None:
        out = np.empty(n, dtype=_np_dtype(c))
    assert out.dtype == _np_dtype(c) and out.size == n and out.flags.c_contiguous
    offset = 1.0 if kind in ("g1", "g2", "gf") else 0.0
    fn = lib.synth_normal_f32 if c.dtype == FP32 else lib.synth_normal_bf16
    fn(c.seed, tensor_id(kind, layer, expert), 0, n, 0.02, offset, out.ctypes.data)
    return out.reshape(shape)


def gen_weights(c: ModelConfig,
                expert_alloc: Optional[Callable[[Tuple[int, ...]], np.ndarray]] = None) -> dict:
    """All weights of config `c` as numpy arrays (fp32, or uint16 holding bf16 bits).

    `expert_alloc(shape)` may supply the storage for expert blobs (e.g. views of pinned
    host memory); the default is ordinary numpy memory."""
    W: dict = {}
    for k, shp in global_shapes(c).items():
        W[k] = gen_tensor(c, k, shp)
    W["layers"] = []
    for l in range(c.n_layers):
        L = {k: gen_tensor(c, k, shp, l) for k, shp in layer_shapes(c, l).items()}
        if c.is_moe:
            L["experts"] = []
            for e in range(c.n_experts):
                E = {}
                for k, shp in expert_shapes(c).items():
                    out = None
                    if expert_alloc is not None:
                        out = expert_alloc(shp).reshape(-1)
                    E[k] = gen_tensor(c, k, shp, l, e, out=out)
                L["experts"].append(E)
        W["layers"].append(L)
    return W


def zero_adapters(c: ModelConfig, W: dict) -> None:
    """Set every adapter B-matrix to zero in place (invariant I3: p == h)."""
    for L in W["layers"]:
        for k in ("Bq", "Bk", "Bv", "Bo", "Bg", "Bu", "Bd"):
            if k in L:
                L[k][...] = 0
    if "lm_B" in W:
        W["lm_B"][...] = 0


def gen_prompt(c: ModelConfig, length: int, seq: int = 0, seed: int = 1000) -> np.ndarray:
    lib = _load()
    out = np.empty(length, dtype=np.int32)
    lib.synth_tokens(seed, seq, length, c.vocab, out.ctypes.data)
    return out


def gen_logit_script(c: ModelConfig, n: int, alpha: float, seq: int = 0, seed: int = 2000):
    """(full_tok[n], draft_tok[n]) — forced-acceptance script, SURVEY §8(d)."""
    lib = _load()
    f = np.empty(n, dtype=np.int32)
    g = np.empty(n, dtype=np.int32)
    lib.synth_logit_script(seed, seq, n, c.vocab, float(alpha), f.ctypes.data, g.ctypes.data)
    return f, g


def gen_router_script(c: ModelConfig, n_steps: int, rho: float, pi: float, seed: int = 3000):
    """(actual[n_steps, N, 2], predicted[n_steps, N, 2]) — seeded routing script."""
    lib = _load()
    a = np.empty((n_steps, c.n_layers, 2), dtype=np.int32)
    p = np.empty((n_steps, c.n_layers, 2), dtype=np.int32)
    lib.synth_router_script(seed, 0, n_steps, c.n_layers, c.n_experts, float(rho), float(pi),
                            a.ctypes.data, p.ctypes.data)
    return a, p


def bf16_bits_to_f32(a: np.ndarray) -> np.ndarray:
    """Widen stored bf16 bit patterns to fp32 (exact)."""
    return (a.astype(np.uint32) << 16).view(np.float32)


def as_f32(c: ModelConfig, a: np.ndarray) -> np.ndarray:
    return a if c.dtype == FP32 else bf16_bits_to_f32(a)
