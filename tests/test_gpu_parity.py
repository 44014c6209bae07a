"""GPU parity: the CUDA path (through the C ABI) vs the CPU oracle, element by element on the same
seeded inputs.  Tolerances are BASELINE.json's: integer work bit-exact (except where the ORACLE's
top-2 margin < 1e-3), fp32 tiny config rel-L2 <= 1e-4, bf16 hidden rel-L2 <= 1e-2 and logits
max-abs <= 5e-2.  Every test here needs a B200 and fails loudly without one."""
import numpy as np
import pytest

import m2r2_synth as S
import paper_2502_02040_b200 as M
from oracle import Oracle
from tests.parity import MARGIN, check_logits, compare_decode_step, tolerances
from tests.refs import rel_l2

# Two CUDA implementations of the same step (persistent fused kernel vs per-operation kernels) are
# cross-checked on bf16 models.  The fused kernel feeds activations to the tensor pipe as bf16
# hi + lo pairs (relative error <= 2^-17 per element), the
# per-operation kernels use fp32 activations, so they agree to a few 1e-5, not to fp32 rounding.  Two RUNS of the
# same implementation differ as well: split-K partial sums are added onto the residual with fp32 atomics in launch
# order (1e-7), and where such a difference crosses a bf16 rounding boundary of a cached K/V element that element
# moves by 2^-9; over a few layers the logits of two engines agree to 1-2e-4 (observed), so the bound is 5e-4.
# (Oracle parity keeps BASELINE.json's tolerances; this constant is not used there.)
XIMPL_TOL = 5e-4

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests selected without a CUDA device: refusing to skip silently"
    cap = torch.cuda.get_device_capability(0)
    assert cap[0] == 10, "libm2r2.so holds sm_100a code only; found sm_%d%d" % cap


def _pair(cfg, W=None, exit_heads=True):
    W = W if W is not None else S.gen_weights(cfg)
    return M.Engine(cfg, W, exit_heads=exit_heads), Oracle(cfg, W), W


def _decode_parity(cfg, P, n_steps, W=None, check_kv=True):
    eng, orc, W = _pair(cfg, W)
    prompt = S.gen_prompt(cfg, P)
    fo = orc.prefill(prompt)
    fe = int(eng.prefill(prompt)[0])
    check_logits(cfg, eng.debug_read(M.DBG_LOGITS, (P - 1) % 8), orc.logits(), "prefill logits")
    assert fe == fo or orc.margin() < MARGIN
    worst = 0.0
    for s in range(n_steps):
        tok_in = orc.pending
        to, exo = orc.decode_step()
        te, exe = eng.decode_step(force_tokens=[tok_in], want_exit=True)   # teacher forcing (Q23)
        worst = max(worst, compare_decode_step(cfg, eng, orc, M))
        assert int(te[0]) == to or orc.margin() < MARGIN, (s, te, to, orc.margin())
        for j in range(len(cfg.gates)):
            if cfg.gates[j] <= cfg.accel_end_layer:
                check_logits(cfg, eng.debug_read(M.DBG_EXIT_LOGITS, j), orc.exit_logits(j), "exit logits %d" % j)
                top2 = np.sort(orc.exit_logits(j))[-2:]
                assert int(exe[0][j]) == int(exo[j]) or top2[1] - top2[0] < MARGIN
        assert eng.get_stats()["kv_len"][0] == orc.kv_len
    if check_kv:
        T = orc.kv_len
        tol = 0 if cfg.dtype == S.FP32 else 1e-2
        for i in range(cfg.n_layers):
            for v in (False, True):
                got = eng.kcache(i, T, v=v)
                want = (orc.vcache(i) if v else orc.kcache(i))[:T]
                assert rel_l2(got, want) <= max(tol, 1e-5), (i, v, rel_l2(got, want))
    eng.close()
    return worst


def test_c1_dual_stream_decode_matches_oracle():
    """BASELINE configs[0]: prefill 32 then 32 decode steps; h_i, p_i, logits, tokens, exit tokens, KV."""
    worst = _decode_parity(S.config_c1(), 32, 32)
    assert worst <= 1e-4


def test_c1_tokens_equal_golden_greedy_stream():
    """Free-running (no teacher forcing) greedy decode on the GPU reproduces the oracle-written
    golden token stream (tests/golden/c1_tokens.txt) unless an oracle margin is < 1e-3."""
    import os
    cfg = S.config_c1()
    gold = [int(t) for t in open(os.path.join(os.path.dirname(__file__), "golden", "c1_tokens.txt")).read().split("\n")[2].split()]
    eng, orc, _ = _pair(cfg)
    prompt = S.gen_prompt(cfg, 32)
    toks = [int(eng.prefill(prompt)[0])]
    orc.prefill(prompt)
    ok = orc.margin() >= MARGIN
    for _ in range(31):
        toks.append(int(eng.decode_step()[0]))
        orc.decode_step()
        ok = ok and orc.margin() >= MARGIN
        if not ok:
            break
    n = len(toks)
    assert toks[:n - (0 if ok else 1)] == gold[:n - (0 if ok else 1)]
    eng.close()


@pytest.mark.parametrize("P", [1, 7, 37])
def test_small_bf16_decode_matches_oracle(P):
    """bf16 storage, head_dim 96, ragged sizes (d_ff 1000, vocab 3001), two gates; short/ragged prompts."""
    worst = _decode_parity(S.config_small_bf16(), P, 6)
    assert worst <= 1e-2


def test_accel_disabled_matches_oracle_and_h_is_unchanged():
    """I2 on the GPU: the slow stream with the accelerated stream on equals the slow stream with it off.
    Equal to fp32 summation order, not bit for bit: the fused kernel's split-K phases add their partial
    sums into the residual with red.global.add.f32, whose order varies from launch to launch
    (DESIGN.md §6.2).  A dependence of h on p would show up at the 1e-2 level (adapters are ~5% of a
    projection), an order of magnitude above this bound, and the slow path is the same code in both engines."""
    cfg_on = S.config_small_bf16()
    cfg_off = S.config_small_bf16(accel_enabled=False, gates=(), accel_end_layer=0)
    W = S.gen_weights(cfg_on)
    e_on, e_off = M.Engine(cfg_on, W), M.Engine(cfg_off, W)
    prompt = S.gen_prompt(cfg_on, 19)
    assert e_on.prefill(prompt)[0] == e_off.prefill(prompt)[0]
    for _ in range(4):
        a, b = e_on.decode_step(), e_off.decode_step()
        assert a[0] == b[0]
        for i in range(cfg_on.n_layers + 1):
            assert rel_l2(e_on.debug_read(M.DBG_H, i), e_off.debug_read(M.DBG_H, i)) <= 1e-3, i
    e_on.close()
    e_off.close()


def test_gate_reset_and_zero_adapter_invariants_on_gpu():
    """I3/I4 on the GPU: with zero adapters and S = all heads, p_i == h_i (to fp32 rounding).
    Run with fp32 storage: with a bf16 cache the slow stream reads its own K[t], V[t] back
    ROUNDED while p keeps k^_t, v^_t in fp32 (Q20), so the identity only holds to
    bf16 rounding there."""
    cfg = S.config_small_bf16(accel_heads=(0, 1, 2, 3), dtype=S.FP32)
    W = S.gen_weights(cfg)
    S.zero_adapters(cfg, W)
    eng = M.Engine(cfg, W)
    eng.prefill(S.gen_prompt(cfg, 9))
    eng.decode_step()
    for i in range(cfg.n_layers + 1):
        assert rel_l2(eng.debug_read(M.DBG_P, i), eng.debug_read(M.DBG_H, i)) <= 1e-5, i
    eng.close()


# ------------------------------------------------------------------ self-speculative decoding
def _c1_selfspec_run(cfg, W, gamma, prompt_seed):
    """-> (tokens compared, tied).  Stops at the first step on which the ORACLE's own margin is < 1e-3."""
    eng, orc = M.Engine(cfg, W), Oracle(cfg, W)
    plain = Oracle(cfg, W)
    prompt = S.gen_prompt(cfg, 32, seed=1000 + prompt_seed)
    first = orc.prefill(prompt)
    if orc.margin() < MARGIN:
        eng.close()
        return 0, True
    assert int(eng.prefill(prompt)[0]) == first
    stream_plain = [plain.prefill(prompt)]
    emitted = [first]
    tie = False
    while len(emitted) < 33:
        acc_o, _ = orc.spec_step(gamma)
        tie = orc.step_margin() < MARGIN
        acc_e, n_e = eng.spec_step(gamma)
        if tie:
            break
        assert acc_e[0][:n_e[0]].tolist() == acc_o
        assert (acc_e[0][n_e[0]:] == -1).all()
        assert eng.get_stats()["kv_len"][0] == orc.kv_len
        check_logits(cfg, eng.debug_read(M.DBG_LOGITS, gamma), orc.logits(), "verify logits row gamma")
        emitted += acc_o
        st, so = eng.get_stats(), orc.stats()
        assert (st["drafted"], st["accepted"], st["emitted"]) == (so["drafted"], so["accepted"], so["emitted"])
    while len(stream_plain) < len(emitted):
        stream_plain.append(plain.decode_step()[0])
    assert emitted == stream_plain[:len(emitted)]      # lossless up to the tie
    eng.close()
    return len(emitted) - 1, tie


@pytest.mark.parametrize("gamma", [0, 1, 3, 6])
def test_c1_selfspec_matches_oracle_and_is_lossless(gamma):
    """a10-a12: accepted tokens, accepted lengths, kv_len bit-exact vs the oracle; emitted stream ==
    plain greedy stream (lossless).  A near-tie in the oracle (margin < 1e-3, Q23) ends the
    comparison for that prompt only; further prompts are run until at least 32 tokens have been compared, so
    the test cannot pass vacuously."""
    cfg = S.config_c1()
    W = S.gen_weights(cfg)
    total = 0
    for prompt_seed in range(6):
        n, tied = _c1_selfspec_run(cfg, W, gamma, prompt_seed)
        total += n
        if total >= 32:
            break
    assert total >= 32, total


@pytest.mark.parametrize("alpha", [0.5, 0.9])
@pytest.mark.parametrize("gamma", [2, 4, 6])
def test_bf16_selfspec_closed_form_acceptance(alpha, gamma):
    """I10 on the GPU: under the logit script the accepted lengths are computable from the seed
    alone: n_accepted - 1 = min(gamma, first j with g != f); kv_len is the running sum; the
    emitted stream is exactly f.  Then KV[0..kv_len) equals the oracle's after rollback (I8)."""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True)
    eng, orc, _ = _pair(cfg)
    P, n_script = 21, 120
    f, g = S.gen_logit_script(cfg, n_script, alpha)
    prompt = S.gen_prompt(cfg, P)
    eng.set_logit_script(f, g, P)
    orc.set_logit_script(f, g, P)
    assert int(eng.prefill(prompt)[0]) == f[0] == orc.prefill(prompt)
    pos = P          # position of the pending token
    emitted = 1
    while emitted + gamma + 1 < 100:
        acc_e, n_e = eng.spec_step(gamma)
        acc_o, _ = orc.spec_step(gamma)
        n = int(n_e[0])
        a = 0
        while a < gamma and g[pos + 1 + a - P] == f[pos + 1 + a - P]:
            a += 1
        assert n == a + 1 == len(acc_o)
        assert acc_e[0][:n].tolist() == f[pos + 1 - P: pos + 1 - P + n].tolist() == acc_o
        pos += n
        emitted += n
        assert eng.get_stats()["kv_len"][0] == pos == orc.kv_len
    for i in range(cfg.n_layers):
        assert rel_l2(eng.kcache(i, pos), orc.kcache(i)[:pos]) <= 1e-2
        assert rel_l2(eng.kcache(i, pos, v=True), orc.vcache(i)[:pos]) <= 1e-2
    # continuing with plain decode after rollback reproduces the scripted stream
    for _ in range(3):
        t = int(eng.decode_step()[0])
        assert t == f[pos + 1 - P]
        pos += 1
    eng.close()


def test_spec_step_zero_equals_decode_step_on_gpu():
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2)
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    prompt = S.gen_prompt(cfg, 11)
    a.prefill(prompt)
    b.prefill(prompt)
    for _ in range(3):
        ta = int(a.decode_step()[0])
        acc, n = b.spec_step(0)
        assert n[0] == 1 and int(acc[0][0]) == ta
        assert rel_l2(a.debug_read(M.DBG_LOGITS, 0), b.debug_read(M.DBG_LOGITS, 0)) <= XIMPL_TOL
    a.close()
    b.close()


@pytest.mark.parametrize("gamma", [1, 4, 7])
def test_verify_rows_on_tensor_cores_match_row_major_kernels(gamma):
    """a11: the skinny tensor-core GEMM on the fragment-major weights (<= 8 rows; verify pass and prefill
    chunks) against the row-major fp32-FMA kernels of the same library: prefill + verify logits of every row,
    accepted tokens and K/V after rollback (ragged d_ff 1000, vocab 3001, head_dim 96).  Both implementations
    are held to the oracle by the other tests; here they are held to each other.  The bound is not fp32
    rounding: products with bf16 hi + lo operands differ from fp32 FMAs by ~1e-6, which flips the bf16
    rounding of about one K/V element in a thousand (measured 1.2e-4 rel-L2 on the layer-0 cache, 1.4e-3 on
    layer 5, 3.8e-4 on the logits).  Tokens are forced by the logit script so that a near-tie cannot
    desynchronise the two engines."""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True)
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    b.set_fused(False)          # per-operation kernels everywhere, row-major weights
    P = 29
    f, g = S.gen_logit_script(cfg, 120, 0.7)
    a.set_logit_script(f, g, P)
    b.set_logit_script(f, g, P)
    prompt = S.gen_prompt(cfg, P)
    assert int(a.prefill(prompt)[0]) == int(b.prefill(prompt)[0]) == f[0]
    assert rel_l2(a.debug_read(M.DBG_LOGITS, (P - 1) % 8), b.debug_read(M.DBG_LOGITS, (P - 1) % 8)) <= 2e-3
    for _ in range(4):
        acc_a, n_a = a.spec_step(gamma)
        acc_b, n_b = b.spec_step(gamma)
        assert n_a[0] == n_b[0] and acc_a[0][:n_a[0]].tolist() == acc_b[0][:n_b[0]].tolist()
        for j in range(gamma + 1):
            assert rel_l2(a.debug_read(M.DBG_LOGITS, j), b.debug_read(M.DBG_LOGITS, j)) <= 2e-3, j
    T = a.get_stats()["kv_len"][0]
    assert T == b.get_stats()["kv_len"][0]
    for i in range(cfg.n_layers):
        assert rel_l2(a.kcache(i, T), b.kcache(i, T)) <= 5e-3
        assert rel_l2(a.kcache(i, T, v=True), b.kcache(i, T, v=True)) <= 5e-3
    a.close()
    b.close()


# ------------------------------------------------------------------ batch (C4 structure, reduced)
def test_batched_selfspec_per_sequence_divergence():
    """B=3 sequences, per-sequence scripts => per-sequence accepted lengths and kv_len diverge; each
    sequence must equal its own single-sequence oracle."""
    B, P, gamma = 3, 13, 4
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True, max_batch=B)
    W = S.gen_weights(cfg)
    eng = M.Engine(cfg, W)
    orcs = [Oracle(cfg, W) for _ in range(B)]
    prompts = np.stack([S.gen_prompt(cfg, P, seq=b) for b in range(B)])
    scripts = [S.gen_logit_script(cfg, 80, 0.7, seq=b) for b in range(B)]
    eng.set_logit_script(np.stack([s[0] for s in scripts]), np.stack([s[1] for s in scripts]), P)
    for b in range(B):
        orcs[b].set_logit_script(scripts[b][0], scripts[b][1], P)
    first = eng.prefill(prompts)
    for b in range(B):
        assert int(first[b]) == orcs[b].prefill(prompts[b])
    for _ in range(8):
        acc, n = eng.spec_step(gamma)
        kv = eng.get_stats()["kv_len"]
        for b in range(B):
            ao, _ = orcs[b].spec_step(gamma)
            assert acc[b][:n[b]].tolist() == ao, (b, acc[b], ao)
            assert kv[b] == orcs[b].kv_len
    assert len(set(eng.get_stats()["kv_len"])) > 1, "scripts should make kv_len diverge"
    for b in range(B):
        T = orcs[b].kv_len
        assert rel_l2(eng.kcache(0, T, b=b), orcs[b].kcache(0)[:T]) <= 1e-2
        assert rel_l2(eng.kcache(cfg.n_layers - 1, T, b=b, v=True), orcs[b].vcache(cfg.n_layers - 1)[:T]) <= 1e-2
    eng.close()


def test_batched_decode_hidden_states_per_sequence():
    B, P = 4, 10
    cfg = S.config_small_bf16(max_batch=B)
    W = S.gen_weights(cfg)
    eng = M.Engine(cfg, W)
    orcs = [Oracle(cfg, W) for _ in range(B)]
    prompts = np.stack([S.gen_prompt(cfg, P, seq=b) for b in range(B)])
    eng.prefill(prompts)
    for b in range(B):
        orcs[b].prefill(prompts[b])
    for _ in range(3):
        forced = [orcs[b].pending for b in range(B)]
        for b in range(B):
            orcs[b].decode_step()
        eng.decode_step(force_tokens=forced)
        for b in range(B):
            compare_decode_step(cfg, eng, orcs[b], M, b=b)
    eng.close()


# ------------------------------------------------------------------ MoE + ahead-of-time expert loading
def _moe_pair(cfg):
    eng = M.Engine(cfg)
    W = S.gen_weights(cfg, expert_alloc=eng.pinned_expert_alloc())
    eng.load_weights(W)
    return eng, Oracle(cfg, W), W


@pytest.mark.parametrize("policy", [M.POLICY_FIXED, M.POLICY_LRU, M.POLICY_LRU_AOT, M.POLICY_LRU_RANDOM, M.POLICY_LRU_PREV])
def test_small_moe_decode_matches_oracle(policy):
    """a13-a17 and the five expert-loading strategies of PAPER.md L242: hidden states, routed / predicted expert
    indices, router weights and the cache counters (hits, misses, prefetched, on-demand) equal the oracle's logical
    LRU model (I15, I22, I23), natural routing."""
    cfg = S.config_small_moe()
    eng, orc, _ = _moe_pair(cfg)
    eng.set_policy(policy)
    orc.set_policy(policy)
    prompt = S.gen_prompt(cfg, 12)
    assert int(eng.prefill(prompt)[0]) == orc.prefill(prompt) or orc.margin() < MARGIN
    for s in range(10):
        tok_in = orc.pending
        orc.decode_step()
        eng.decode_step(force_tokens=[tok_in])
        compare_decode_step(cfg, eng, orc, M)
        ri = eng.debug_read(M.DBG_ROUTE_IDX).reshape(cfg.n_layers, cfg.top_k).astype(np.int32)
        assert np.array_equal(ri, orc.route_idx()), (s, ri, orc.route_idx())
        assert np.allclose(eng.debug_read(M.DBG_ROUTE_W).reshape(cfg.n_layers, cfg.top_k), orc.route_w(), atol=2e-3)
        if policy >= M.POLICY_LRU_AOT:
            pi = eng.debug_read(M.DBG_PRED_IDX).reshape(cfg.n_layers, cfg.top_k).astype(np.int32)
            po = orc.pred_idx()
            mask = po >= 0
            assert np.array_equal(pi[mask], po[mask]), (s, pi, po)
        st, so = eng.get_stats(), orc.stats()
        assert (st["expert_hits"], st["expert_misses"], st["expert_prefetched"], st["expert_on_demand"]) == \
               (so["expert_hits"], so["expert_misses"], so["prefetched"], so["on_demand"]), (s, st, so)
    one = 3 * cfg.d_ff_expert * cfg.d_model * 2
    st = eng.get_stats()
    assert st["h2d_bytes"] == (st["expert_prefetched"] + st["expert_on_demand"]) * one
    eng.close()


@pytest.mark.parametrize("rho,pi", [(0.25, 0.9), (0.0, 1.0)])
def test_small_moe_router_script_counters(rho, pi):
    """Scripted routing (seeded 'random logits', BASELINE configs[4]): with pi = 1 every targeted layer
    has zero misses; counters equal the oracle's; output h does not depend on the policy (I14)."""
    cfg = S.config_small_moe()
    eng, orc, _ = _moe_pair(cfg)
    P, n = 8, 24
    act, pred = S.gen_router_script(cfg, n + P + 1, rho, pi)
    eng.set_policy(M.POLICY_LRU_AOT)
    orc.set_policy(2)
    eng.set_router_script(act, pred, 0)
    orc.set_router_script(act, pred, 0)
    prompt = S.gen_prompt(cfg, P)
    eng.prefill(prompt)
    orc.prefill(prompt)
    for s in range(n):
        tok_in = orc.pending
        orc.decode_step()
        eng.decode_step(force_tokens=[tok_in])
        ri = eng.debug_read(M.DBG_ROUTE_IDX).reshape(cfg.n_layers, cfg.top_k).astype(np.int32)
        assert np.array_equal(ri, act[P + s]), (s, ri, act[P + s])
    compare_decode_step(cfg, eng, orc, M)
    st, so = eng.get_stats(), orc.stats()
    assert (st["expert_hits"], st["expert_misses"], st["expert_prefetched"], st["expert_on_demand"]) == \
           (so["expert_hits"], so["expert_misses"], so["prefetched"], so["on_demand"])
    assert st["expert_hits"] + st["expert_misses"] == cfg.top_k * cfg.n_layers * n
    eng.close()


def test_moe_explicit_prefetch_pairs_then_hits():
    """m2r2_moe_prefetch(pairs): prefetching exactly the experts the script will route makes them hits."""
    cfg = S.config_small_moe()
    eng, _, _ = _moe_pair(cfg)
    P = 5
    act, _ = S.gen_router_script(cfg, P + 4, 0.0, 1.0)
    eng.set_policy(M.POLICY_LRU)
    eng.set_router_script(act, act, 0)
    eng.prefill(S.gen_prompt(cfg, P))
    pairs = [(L, int(e)) for L in range(cfg.n_layers) for e in act[P][L]]
    n = eng.moe_prefetch(pairs=pairs)
    assert 0 <= n <= len(pairs)
    eng.decode_step()
    st = eng.get_stats()
    assert st["expert_misses"] == 0 and st["expert_hits"] == cfg.top_k * cfg.n_layers
    assert st["expert_prefetched"] == n
    eng.close()


# ------------------------------------------------------------------ error behaviour on a live context
def test_error_codes_on_live_context():
    cfg = S.config_c1()
    eng = M.Engine(cfg, S.gen_weights(cfg))
    with pytest.raises(M.M2R2Error) as e:
        eng.B = 1
        eng.decode_step()
    assert e.value.code == M.BAD_STATE
    with pytest.raises(M.M2R2Error) as e:
        eng.prefill(np.full(4, cfg.vocab, dtype=np.int32))
    assert e.value.code == M.INVALID_ARG
    with pytest.raises(M.M2R2Error) as e:
        eng.prefill(np.zeros(cfg.max_seq + 1, dtype=np.int32))
    assert e.value.code == M.INVALID_ARG
    eng.prefill(S.gen_prompt(cfg, cfg.max_seq - 2))
    with pytest.raises(M.M2R2Error) as e:
        eng.spec_step(3)
    assert e.value.code == M.CAPACITY
    kv = eng.get_stats()["kv_len"][0]
    eng.decode_step()
    eng.decode_step()
    assert eng.get_stats()["kv_len"][0] == kv + 2 == cfg.max_seq
    with pytest.raises(M.M2R2Error) as e:
        eng.decode_step()
    assert e.value.code == M.CAPACITY
    with pytest.raises(M.M2R2Error) as e:
        eng.spec_step(8)
    assert e.value.code == M.INVALID_ARG
    with pytest.raises(M.M2R2Error) as e:
        eng.moe_prefetch(0)
    assert e.value.code == M.UNSUPPORTED
    eng.close()


def test_dead_positions_do_not_leak_after_rollback():
    """I8 on the GPU: K/V at positions >= kv_len are dead: running a spec step that rejects drafts and
    then decoding gives the same tokens as an engine that never drafted."""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2)
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    P = 17
    f, g = S.gen_logit_script(cfg, 60, 0.0)      # alpha = 0: every draft is rejected
    for e in (a, b):
        e.set_logit_script(f, g, P)
        e.prefill(S.gen_prompt(cfg, P))
    for s in range(5):
        acc, n = a.spec_step(5)
        assert n[0] == 1
        t = b.decode_step()
        assert int(acc[0][0]) == int(t[0]) == f[s + 1]
        assert rel_l2(a.debug_read(M.DBG_LOGITS, 0), b.debug_read(M.DBG_LOGITS, 0)) <= XIMPL_TOL
    a.close()
    b.close()


# ------------------------------------------------------------------ full size (BASELINE.json configs[1] / [2]), the launch configuration bench.py times
def test_c2_full_size_fused_step_matches_oracle_at_short_context():
    """The 3.8B-class model itself (32 layers, d 3072, 32 x 96 heads, FFN 8192, vocab 32064, gates 8/16/24,
    both streams in every layer), through the same persistent fused kernel and launch configuration that
    bench.py times.  The oracle needs 0.35 s per token at this size, so the context is short (prompt 6,
    three teacher-forced decode steps): every h_i and p_i of every layer (rel-L2 <= 1e-2), the final logits
    (max-abs <= 5e-2), the greedy token and the three exit tokens (exact unless the oracle's margin < 1e-3)."""
    cfg = S.config_c2()
    W = S.gen_weights(cfg)
    eng, orc = M.Engine(cfg, W, exit_heads=True), Oracle(cfg, W)
    prompt = S.gen_prompt(cfg, 6)
    fo, fe = orc.prefill(prompt), int(eng.prefill(prompt)[0])
    check_logits(cfg, eng.debug_read(M.DBG_LOGITS, 5), orc.logits(), "prefill logits")
    assert fe == fo or orc.margin() < MARGIN
    for s in range(3):
        tok_in = orc.pending
        to, exo = orc.decode_step()
        te, exe = eng.decode_step(force_tokens=[tok_in], want_exit=True)
        worst = compare_decode_step(cfg, eng, orc, M)
        assert worst <= 1e-2
        assert int(te[0]) == to or orc.margin() < MARGIN, (s, te, to, orc.margin())
        for j in range(len(cfg.gates)):
            check_logits(cfg, eng.debug_read(M.DBG_EXIT_LOGITS, j), orc.exit_logits(j), "exit logits %d" % j)
            top2 = np.sort(orc.exit_logits(j))[-2:]
            assert int(exe[0][j]) == int(exo[j]) or top2[1] - top2[0] < MARGIN
    assert eng.get_stats()["kv_len"][0] == orc.kv_len == 9
    eng.close()
    orc.close()


def test_c3_full_size_long_context_properties():
    """Full size at the context bench.py runs (prompt 512), where the oracle is too slow to follow: properties
    that hold at any size.  (i) the fused kernel and the per-operation kernels of the same library agree on
    the decode logits (two CUDA implementations with different layouts, split-K orders and attention paths);
    (ii) under the logit script self-speculation emits exactly the scripted stream and the accepted lengths
    follow the closed form (I10), with the draft passes in the fused kernel and the verify pass on the
    tensor-core GEMM; (iii) continuing with plain decode after the rollbacks reproduces the stream (I8)."""
    cfg = S.config_c3()
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    b.set_fused(False)
    P, gamma, alpha = 512, 4, 0.7
    prompt = S.gen_prompt(cfg, P)
    ta, tb = int(a.prefill(prompt)[0]), int(b.prefill(prompt)[0])
    la, lb = a.debug_read(M.DBG_LOGITS, (P - 1) % 8), b.debug_read(M.DBG_LOGITS, (P - 1) % 8)
    assert float(np.max(np.abs(la - lb))) <= 5e-2 and rel_l2(la, lb) <= 5e-3
    margin = np.sort(lb)[-1] - np.sort(lb)[-2]
    assert ta == tb or margin < 5e-2
    for _ in range(2):
        b_tok = b.decode_step()
        a_tok = a.decode_step()
        la, lb = a.debug_read(M.DBG_LOGITS, 0), b.debug_read(M.DBG_LOGITS, 0)
        if int(a_tok[0]) != int(b_tok[0]):
            break   # a near-tie desynchronised the free-running engines: the logits check above already passed
        assert float(np.max(np.abs(la - lb))) <= 5e-2 and rel_l2(la, lb) <= 5e-3
    # (ii) + (iii) on the fused engine
    f, g = S.gen_logit_script(cfg, 200, alpha)
    a.set_logit_script(f, g, P)
    assert int(a.prefill(prompt)[0]) == f[0]
    pos, emitted = P, 1
    while emitted + gamma + 1 < 60:
        acc, n = a.spec_step(gamma)
        n = int(n[0])
        k = 0
        while k < gamma and g[pos + 1 + k - P] == f[pos + 1 + k - P]:
            k += 1
        assert n == k + 1
        assert acc[0][:n].tolist() == f[pos + 1 - P: pos + 1 - P + n].tolist()
        pos += n
        emitted += n
        assert a.get_stats()["kv_len"][0] == pos
    for _ in range(3):
        assert int(a.decode_step()[0]) == f[pos + 1 - P]
        pos += 1
    # (iv) the verify pass at full width and this context: the ring GEMMs with RMSNorm, RoPE + KV append and the split merge
    # absorbed (engine a) against the per-operation kernels (engine b: row-major fp32-FMA GEMV, separate norm / RoPE /
    # merge kernels) on the same scripted steps: logits of every verify row, and the K/V the pass left in the cache
    b.set_logit_script(f, g, P)
    assert int(a.prefill(prompt)[0]) == f[0] and int(b.prefill(prompt)[0]) == f[0]
    for _ in range(2):
        acc_a, n_a = a.spec_step(gamma)
        acc_b, n_b = b.spec_step(gamma)
        assert int(n_a[0]) == int(n_b[0]) and acc_a[0][:int(n_a[0])].tolist() == acc_b[0][:int(n_b[0])].tolist()
        for j in range(gamma + 1):
            la, lb = a.debug_read(M.DBG_LOGITS, j), b.debug_read(M.DBG_LOGITS, j)
            assert float(np.max(np.abs(la - lb))) <= 5e-2 and rel_l2(la, lb) <= 5e-3, (j, float(np.max(np.abs(la - lb))), rel_l2(la, lb))
    T = a.get_stats()["kv_len"][0]
    assert T == b.get_stats()["kv_len"][0] and T > P
    for layer in (0, cfg.n_layers // 2, cfg.n_layers - 1):
        for v in (False, True):
            ka, kb = a.kcache(layer, T, v=v), b.kcache(layer, T, v=v)
            assert rel_l2(ka[P:], kb[P:]) <= 1e-2, (layer, v, rel_l2(ka[P:], kb[P:]))   # the rows the verify passes appended
    a.close()
    b.close()


def _first_steps_stress(cycles):
    """-> number of (cycle, step, layer) checks that exceeded the bound, and the worst error"""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2)
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 11)
    toks = [5, 77, 1234]
    r0 = M.Engine(cfg, W)
    r0.set_fused(False)
    r0.prefill(prompt)
    ref = []
    for s in range(3):
        r0.decode_step(force_tokens=[toks[s]])
        ref.append([r0.debug_read(M.DBG_H, i).copy() for i in range(cfg.n_layers + 1)])
    r0.close()
    bad, worst = 0, 0.0
    for cyc in range(cycles):
        a = M.Engine(cfg, W)
        a.prefill(prompt)
        for s in range(3):
            a.decode_step(force_tokens=[toks[s]])
            for i in range(cfg.n_layers + 1):
                e = rel_l2(a.debug_read(M.DBG_H, i), ref[s][i])
                worst = max(worst, e)
                bad += e > 3e-3
        a.close()
    return bad, worst


def test_ring_race_guard_under_the_padded_scratch_layout():
    """The write-after-read race on the weight ring fired about once per ten launches, but only with
    the adapter scratch padded to one 128-byte line per item; the committed layout is dense and never showed it.
    This test therefore runs the stress on a VARIANT BUILD of the library with that padded layout
    (-DM2R2_PAD_SCRATCH): the committed `release_stage` must hold there.  With M2R2_RACE_DEMO=1 in the environment
    it also builds the variant whose `release_stage` is the plain arrive (-DM2R2_PLAIN_ARRIVE) and requires the
    stress to FAIL on it, i.e. that this test can see the race at all (recorded in profiles/r2_ring_race_guard.md)."""
    import os
    from paper_2502_02040_b200 import binding, build
    try:
        binding.use_library(build.build_variant("pad", ["M2R2_PAD_SCRATCH"]))
        bad, worst = _first_steps_stress(40)
        assert bad == 0, (bad, worst)
        if os.environ.get("M2R2_RACE_DEMO"):
            binding.use_library(build.build_variant("padplain", ["M2R2_PAD_SCRATCH", "M2R2_PLAIN_ARRIVE"]))
            bad, worst = _first_steps_stress(100)
            print("plain arrive + padded scratch: %d checks above the bound, worst rel-L2 %.3g" % (bad, worst))
            assert bad > 0, "the unguarded arrive did not reproduce the race on this box"
    finally:
        binding.use_library(None)


def test_fused_first_steps_repeat_across_engine_instances():
    """Stress for timing-dependent errors in the fused kernel: 40 fresh engines of a model whose first two layers
    carry the accelerated stream and whose other layers do not (the C3 structure, where the auxiliary warp
    retires early), each prefilled and stepped three times under teacher forcing, against the per-operation
    kernels of the same library.  The two implementations differ by ~5e-4 here (bf16 K/V rounding flips); a
    ring stage refilled while a warp still reads it (the race `release_stage` closes: it hit
    a third of these cycles once the adapter scratch was padded) shows up as >= 1e-2 on the 16 rows of one warp."""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2)
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 11)
    toks = [5, 77, 1234]
    r0 = M.Engine(cfg, W)
    r0.set_fused(False)
    r0.prefill(prompt)
    ref = []
    for s in range(3):
        r0.decode_step(force_tokens=[toks[s]])
        ref.append([r0.debug_read(M.DBG_H, i).copy() for i in range(cfg.n_layers + 1)])
    r0.close()
    for cyc in range(40):
        a = M.Engine(cfg, W)
        a.prefill(prompt)
        for s in range(3):
            a.decode_step(force_tokens=[toks[s]])
            for i in range(cfg.n_layers + 1):
                e = rel_l2(a.debug_read(M.DBG_H, i), ref[s][i])
                assert e <= 3e-3, (cyc, s, i, e)
        a.close()


@pytest.mark.parametrize("fused", [True, False])
def test_results_do_not_depend_on_uninitialised_device_memory(fused, monkeypatch):
    """The weights arena, the KV cache and the scratch arena are handed to the library uninitialised
    (`torch.empty`).  Each of the three is filled in turn with 0xFF bytes (NaN as bf16 and as fp32, -1 as an
    index), 0x7F bytes (huge finite values) and seeded random bytes before `m2r2_create`; every hidden state
    of both streams must come out as with zero-filled arenas.  A read of memory the library never wrote (a
    padded weight stage the repack skipped, K/V rows past the context, a partial of an empty attention split,
    a padded activation slot) would show up as NaN or as an O(1) error.  The per-operation kernels are
    deterministic, so they must agree bit for bit; the fused kernel's fp32 atomics reorder, so it agrees to
    rounding."""
    import torch
    orig_empty = torch.empty
    state = {"n": 0, "which": -1, "mode": "zero"}

    def poisoned_empty(*a, **k):
        t = orig_empty(*a, **k)
        if t.is_cuda and t.dtype == torch.uint8:
            i = state["n"] % 3   # Engine allocates weights, kv, scratch in this order
            state["n"] += 1
            if i != state["which"] or state["mode"] == "zero":
                t.zero_()
            elif state["mode"] == "rand":
                g = torch.Generator(device=t.device).manual_seed(7)
                t.copy_(torch.randint(0, 256, t.shape, dtype=torch.uint8, device=t.device, generator=g))
            else:
                t.fill_(int(state["mode"], 16))
        return t

    monkeypatch.setattr(torch, "empty", poisoned_empty)
    toks = [5, 77, 1234, 9, 400]

    def run(cfg, W, prompt):
        state["n"] = 0
        e = M.Engine(cfg, W)
        e.set_fused(fused)
        e.prefill(prompt)
        out = []
        for t in toks:
            e.decode_step(force_tokens=[t])
            out.append(np.stack([e.debug_read(M.DBG_H, i) for i in range(cfg.n_layers + 1)] +
                                [e.debug_read(M.DBG_P, i) for i in range(cfg.n_layers + 1)]))
        e.close()
        return out

    for cfg in (S.config_small_bf16(gates=(2,), accel_end_layer=2), S.config_small_bf16()):
        W = S.gen_weights(cfg)
        for plen in (11, 70):
            prompt = S.gen_prompt(cfg, plen)
            state["which"], state["mode"] = -1, "zero"
            ref = run(cfg, W, prompt)
            for which in range(3):
                for mode in ("ff", "7f", "rand"):
                    state["which"], state["mode"] = which, mode
                    out = run(cfg, W, prompt)
                    for s in range(len(toks)):
                        assert np.all(np.isfinite(out[s])), (plen, which, mode, s)
                        if fused:
                            assert rel_l2(out[s], ref[s]) <= XIMPL_TOL, (plen, which, mode, s, rel_l2(out[s], ref[s]))
                        else:
                            assert np.array_equal(out[s], ref[s]), (plen, which, mode, s)
