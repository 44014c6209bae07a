"""m2r2_final_head_noalloc (include/m2r2.h): the final head with its scratch in a static device array of the library —
the one entry point for callers that cannot call cudaMalloc.  Its output is checked against the existing path's final
head (the engine's per-operation kernels: h_N and the logits of the same decode step, read through m2r2_debug_read)
within the tolerances the parity tests use, on calls in a row that share the scratch.

This file is named to be collected LAST (the suite runs with pytest -x: a failure here must not hide other tests) and
passes both alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import m2r2_synth as S
import paper_2502_02040_b200 as M
from tests.parity import check_logits
from tests.refs import rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests selected without a CUDA device: refusing to skip silently"
    cap = torch.cuda.get_device_capability(0)
    assert cap[0] == 10, "libm2r2.so holds sm_100a code only; found sm_%d%d" % cap


def _dev(a):
    """numpy weight (fp32, or uint16 holding bf16 bits) -> CUDA tensor with the same bytes."""
    import torch
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("which", ["c1_fp32", "small_bf16"])
def test_final_head_noalloc_matches_the_engine_on_calls_in_a_row(which):
    import torch
    cfg = S.config_c1() if which == "c1_fp32" else S.config_small_bf16()
    W = S.gen_weights(cfg)
    eng = M.Engine(cfg, W)
    eng.set_fused(False)   # the existing path's final head = the per-operation kernels (same arithmetic, bit for bit)
    eng.prefill(S.gen_prompt(cfg, 19))
    hs, refs = [], []
    for _ in range(3):
        eng.decode_step()
        hs.append(eng.debug_read(M.DBG_H, cfg.n_layers).copy())
        refs.append(eng.debug_read(M.DBG_LOGITS, 0).copy())
    assert rel_l2(refs[0], refs[1]) > 1e-2, "steps must differ for stale scratch to show"
    g_f, w_lm = _dev(W["gf"]), _dev(W["lm_head"])
    d, V = cfg.d_model, cfg.vocab
    h1 = torch.from_numpy(hs[0]).cuda().reshape(1, d)
    h123 = torch.from_numpy(np.stack(hs)).cuda()
    h3 = torch.from_numpy(hs[2]).cuda().reshape(1, d)
    o1 = torch.full((1, V), float("nan"), device="cuda")
    o123 = torch.full((3, V), float("nan"), device="cuda")
    o3 = torch.full((1, V), float("nan"), device="cuda")
    # warm-up call (resolves the scratch address on this device), then free memory must not move: nothing is allocated
    M.final_head_noalloc(h3, g_f, w_lm, o3, cfg.dtype, cfg.rms_eps)
    torch.cuda.synchronize()
    o3.fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # three calls in a row on one stream, no synchronisation between them, different row counts and inputs
    M.final_head_noalloc(h1, g_f, w_lm, o1, cfg.dtype, cfg.rms_eps)
    M.final_head_noalloc(h123, g_f, w_lm, o123, cfg.dtype, cfg.rms_eps)
    M.final_head_noalloc(h3, g_f, w_lm, o3, cfg.dtype, cfg.rms_eps)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory was allocated during the calls"
    got1, got123, got3 = o1.cpu().numpy(), o123.cpu().numpy(), o3.cpu().numpy()
    check_logits(cfg, got1[0], refs[0], "call 1 (1 row)")
    for j in range(3):
        check_logits(cfg, got123[j], refs[j], "call 2 (3 rows), row %d" % j)
    check_logits(cfg, got3[0], refs[2], "call 3 (1 row)")
    # one-row calls launch exactly the engine's kernels on the same inputs: equal bit for bit, stronger than the tolerance
    assert np.array_equal(got1[0], refs[0]) and np.array_equal(got3[0], refs[2])
    eng.close()


def test_final_head_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    V = 16
    for m, d, what in ((M.NOALLOC_MAX_ROWS + 1, 256, "M2R2_NOALLOC_MAX_ROWS"), (1, M.NOALLOC_MAX_D + 8, "M2R2_NOALLOC_MAX_D")):
        h = torch.zeros((m, d), device="cuda")
        g = torch.ones(d, device="cuda")
        w = torch.zeros((V, d), device="cuda")
        o = torch.full((m, V), 7.0, device="cuda")
        with pytest.raises(M.M2R2Error) as ei:
            M.final_head_noalloc(h, g, w, o, M.FP32, 1e-5)
        assert ei.value.code == M.CAPACITY and what in str(ei.value), str(ei.value)
        torch.cuda.synchronize()
        assert bool((o == 7.0).all()), "a rejected call must not touch the output"
    # d not a multiple of 8: invalid argument, not capacity
    h = torch.zeros((1, 100), device="cuda")
    with pytest.raises(M.M2R2Error) as ei:
        M.final_head_noalloc(h, torch.ones(100, device="cuda"), torch.zeros((V, 100), device="cuda"),
                             torch.zeros((1, V), device="cuda"), M.FP32, 1e-5)
    assert ei.value.code == M.INVALID_ARG
    # the largest accepted shape runs
    d = M.NOALLOC_MAX_D
    h = torch.randn((M.NOALLOC_MAX_ROWS, d), device="cuda")
    g = torch.ones(d, device="cuda")
    w = torch.randn((V, d), device="cuda") * 0.01
    o = torch.empty((M.NOALLOC_MAX_ROWS, V), device="cuda")
    M.final_head_noalloc(h, g, w, o, M.FP32, 1e-5)
    torch.cuda.synchronize()
    ref = (h.double() * torch.rsqrt((h.double() ** 2).mean(1, keepdim=True) + 1e-5)) @ w.double().T
    assert rel_l2(o.cpu().numpy(), ref.cpu().numpy()) <= 1e-4
