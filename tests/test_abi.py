"""CPU-side checks of the boundary: libm2r2.so loads, exports every symbol include/m2r2.h declares,
the POD structs of the binding match the header, and argument validation works without a GPU
(no compute call is made here)."""
import ctypes
import os
import re

import pytest

import m2r2_synth as S
import paper_2502_02040_b200 as M
from paper_2502_02040_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "m2r2.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(m2r2_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared_functions()
    assert len(names) >= 17, names
    L = ctypes.CDLL(M.binding._build.build())
    for n in names:
        assert hasattr(L, n), "libm2r2.so does not export %s" % n
    assert sorted(M.EXPORTS) == names


def test_header_names_the_five_north_star_calls():
    names = _declared_functions()
    for n in ("m2r2_load_weights", "m2r2_prefill", "m2r2_decode_step", "m2r2_spec_step", "m2r2_moe_prefetch"):
        assert n in names


def _c_sizeof(struct_name):
    """sizeof(struct) as gcc sees include/m2r2.h."""
    import subprocess
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        src = os.path.join(td, "s.c")
        exe = os.path.join(td, "s")
        open(src, "w").write('#include <stdio.h>\n#include "%s"\nint main(){printf("%%zu", sizeof(%s));return 0;}\n'
                             % (HEADER, struct_name))
        subprocess.check_call(["gcc", "-o", exe, src])
        return int(subprocess.check_output([exe]).decode())


@pytest.mark.parametrize("cname,pystruct", [("m2r2_config", binding.Config), ("m2r2_sizes", binding.Sizes),
                                            ("m2r2_buffers", binding.Buffers), ("m2r2_stats", binding.Stats),
                                            ("m2r2_layer_weights", binding.LayerWeights),
                                            ("m2r2_weight_table", binding.WeightTable)])
def test_binding_struct_sizes_match_header(cname, pystruct):
    assert _c_sizeof(cname) == ctypes.sizeof(pystruct)


def test_header_is_plain_c():
    """The boundary is a C ABI: the header must compile as C (no C++ / torch types)."""
    assert _c_sizeof("m2r2_config") > 0
    src = open(HEADER).read()
    assert 'extern "C"' in src
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    assert "torch" not in code and "std::" not in code and "at::" not in code


@pytest.mark.parametrize("make", [S.config_c1, S.config_c2, S.config_c3, S.config_c4, S.config_c5,
                                  S.config_small_bf16, S.config_small_moe])
def test_query_sizes_host_only(make):
    cfg = make()
    c = M.make_config(cfg)
    sz = M.Sizes()
    assert M.lib().m2r2_query_sizes(ctypes.byref(c), ctypes.byref(sz)) == M.OK
    e = cfg.elt_bytes
    kv = 2 * cfg.n_layers * cfg.max_batch * cfg.n_heads * cfg.max_seq * cfg.head_dim * e
    assert kv <= sz.kv_bytes <= kv + 4096
    # resident weights: at least the dense matrices + embeddings
    per_layer = 4 * cfg.d_model ** 2 + (0 if cfg.is_moe else 3 * cfg.d_model * cfg.d_ff)
    assert sz.weights_bytes >= (cfg.n_layers * per_layer + 2 * cfg.vocab * cfg.d_model) * e
    if cfg.is_moe:
        one = 3 * cfg.d_ff_expert * cfg.d_model * e
        assert sz.expert_cache_bytes >= cfg.n_layers * cfg.cache_slots * one
        assert sz.expert_store_bytes == cfg.n_layers * cfg.n_experts * one
    else:
        assert sz.expert_cache_bytes == 0


def test_c2_sizes_match_survey_byte_model():
    """3.8B layer = 226,492,416 B bf16, LM head = 197,001,216 B, KV = 12,288 B/pos/layer."""
    cfg = S.config_c2()
    assert (4 * cfg.d_model ** 2 + 3 * cfg.d_model * cfg.d_ff) * 2 == 226_492_416
    assert cfg.vocab * cfg.d_model * 2 == 197_001_216
    assert 2 * cfg.d_model * 2 == 12_288


def test_validation_rejects_bad_configs():
    L = M.lib()
    sz = M.Sizes()
    good = M.make_config(S.config_c1())
    assert L.m2r2_query_sizes(ctypes.byref(good), ctypes.byref(sz)) == M.OK
    assert L.m2r2_query_sizes(None, ctypes.byref(sz)) == M.INVALID_ARG
    assert L.m2r2_query_sizes(ctypes.byref(good), None) == M.INVALID_ARG
    for field, val in (("struct_size", 4), ("n_layers", 0), ("d_model", 250), ("head_dim", 48), ("dtype", 7),
                       ("max_batch", 9), ("vocab", 1), ("adapter_rank", 0), ("accel_end_layer", 99)):
        c = M.make_config(S.config_c1())
        setattr(c, field, val)
        assert L.m2r2_query_sizes(ctypes.byref(c), ctypes.byref(sz)) == M.INVALID_ARG, field
    c = M.make_config(S.config_c1())
    c.gates[0] = 9
    assert L.m2r2_query_sizes(ctypes.byref(c), ctypes.byref(sz)) == M.INVALID_ARG
    c = M.make_config(S.config_c1())
    c.accel_heads[0], c.accel_heads[1] = 1, 1     # not strictly increasing
    assert L.m2r2_query_sizes(ctypes.byref(c), ctypes.byref(sz)) == M.INVALID_ARG
    c = M.make_config(S.config_small_moe())
    c.aot_lo[2], c.aot_hi[2] = 1, 3               # a target range must start above its source
    assert L.m2r2_query_sizes(ctypes.byref(c), ctypes.byref(sz)) == M.INVALID_ARG


def test_null_context_calls_return_invalid_arg():
    L = M.lib()
    assert L.m2r2_destroy(None) == M.INVALID_ARG
    assert L.m2r2_reset(None) == M.INVALID_ARG
    assert L.m2r2_decode_step(None, None, None, None) == M.INVALID_ARG
    assert L.m2r2_spec_step(None, 1, None, None) == M.INVALID_ARG
    assert L.m2r2_prefill(None, None, 1, 1, None) == M.INVALID_ARG
    assert L.m2r2_moe_prefetch(None, 0, None, 0) == M.INVALID_ARG
    assert L.m2r2_last_error(None) == b"null context"
    assert b"sm_100a" in L.m2r2_version()


def test_engine_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        M.Engine(S.config_c1())


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (③): no file under the package,
    include/ or m2r2_synth/ mentions the oracle package as an import."""
    for base in ("paper_2502_02040_b200", "m2r2_synth", "include"):
        for dp, _, fns in os.walk(os.path.join(ROOT, base)):
            for fn in fns:
                if fn.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                    src = open(os.path.join(dp, fn)).read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), (dp, fn)
                    assert "m2r2_oracle" not in src, (dp, fn)
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "m2r2_oracle.c")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_2502_02040_b200\b", orc, flags=re.M)
    assert "m2r2.h" not in orc.replace("include/m2r2.h", "")
