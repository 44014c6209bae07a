"""GPU parity at the sizes and on the code paths the kernels actually run ("next round" item 1).

Each test names the branch of the CUDA path it reaches (DESIGN.md §3 has the table).  All comparisons are
against the CPU oracle on the same seeded inputs, with BASELINE.json's tolerances (tests/parity.py)."""
from dataclasses import replace

import numpy as np
import pytest

import m2r2_synth as S
import paper_2502_02040_b200 as M
from oracle import Oracle
from tests.parity import MARGIN, check_hidden, check_logits, compare_decode_step
from tests.refs import rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests selected without a CUDA device: refusing to skip silently"


def _teacher_forced(cfg, P, n_steps, exit_heads=True, check_kv_layers=()):
    W = S.gen_weights(cfg)
    eng, orc = M.Engine(cfg, W, exit_heads=exit_heads), Oracle(cfg, W)
    prompt = S.gen_prompt(cfg, P)
    fo, fe = orc.prefill(prompt), int(eng.prefill(prompt)[0])
    check_logits(cfg, eng.debug_read(M.DBG_LOGITS, (P - 1) % 8), orc.logits(), "prefill logits")
    assert fe == fo or orc.margin() < MARGIN
    worst = 0.0
    for s in range(n_steps):
        tok_in = orc.pending
        to, exo = orc.decode_step()
        te, exe = eng.decode_step(force_tokens=[tok_in], want_exit=True)
        worst = max(worst, compare_decode_step(cfg, eng, orc, M))
        assert int(te[0]) == to or orc.margin() < MARGIN, (s, te, to, orc.margin())
        if exit_heads:
            for j in range(len(cfg.gates)):
                check_logits(cfg, eng.debug_read(M.DBG_EXIT_LOGITS, j), orc.exit_logits(j), "exit logits %d" % j)
                top2 = np.sort(orc.exit_logits(j))[-2:]
                assert int(exe[0][j]) == int(exo[j]) or top2[1] - top2[0] < MARGIN
        assert eng.get_stats()["kv_len"][0] == orc.kv_len
    T = orc.kv_len
    for i in check_kv_layers:
        assert rel_l2(eng.kcache(i, T), orc.kcache(i)[:T]) <= 1e-2
        assert rel_l2(eng.kcache(i, T, v=True), orc.vcache(i)[:T]) <= 1e-2
    st = eng.get_stats()
    eng.close()
    orc.close()
    return worst, st


def test_c2_shaped_long_context_multi_round_attention_staging():
    """C2's attention geometry (32 heads x 96, d 3072) on a 2-layer model, prompt 800, 8 teacher-forced steps:
    the fused kernel runs ns = 4 splits of 200-202 positions each, i.e. MORE than one staging round per split
    (cap = 192 positions at head_dim 96: `attn_phase`'s `r0 > p0` branch), and the O-proj loader merges four
    splits per head.  Every h_i, p_i, the logits, tokens, exit tokens and the K/V cache against the oracle."""
    cfg = replace(S.config_c2(), name="C2-narrow", n_layers=2, d_ff=1024, vocab=2048, max_seq=832,
                  gates=(1,), accel_end_layer=2, seed=0x4D325232 + 21)
    worst, st = _teacher_forced(cfg, 800, 8, check_kv_layers=(0, 1))
    assert worst <= 1e-2
    assert st["kernel_launches"] > 0


@pytest.mark.parametrize("P", [165, 1001])
def test_four_heads_long_context_unstaged_merge(P):
    """n_heads = 4 gives the fused kernel 148 / 4 = 37 CTAs per head, so the number of attention splits is
    bounded by the context: T = 165 -> ns = 6 > MERGE_NS (the looped `combine_slow` of the auxiliary warp, with
    the partials still staged in shared memory); T = 1001 -> ns = 32, whose partials of two heads exceed the
    40 KB staging area (`merge_global`, the unstaged merge of the O-proj loader)."""
    cfg = S.config_small_bf16(max_seq=P + 16)
    worst, _ = _teacher_forced(cfg, P, 4, check_kv_layers=(0, cfg.n_layers - 1))
    assert worst <= 1e-2


@pytest.mark.parametrize("shape", ["c3", "gemma"])
def test_unscripted_selfspec_draft_head_and_lm_adapter_match_oracle(shape):
    """(shape "gemma": SURVEY 8(f) f-4, the structure of `config_gemma7b_class` reduced: 128-wide heads, the draft gate
    after ONE of six layers and a vocabulary 50x the model width, so the LM head dominates the draft as the 256k-row
    head does at full size.)
    a8/a10 on the path C3 runs: bf16 model with a single draft gate and the LM-head adapter, spec_step WITHOUT
    a logit script, so the draft tokens are decided by the fused draft pass itself (PH_HEAD with head_stream = 1:
    `LN_HEAD_P` loader, `lmA`/`lmB` adapter, joff > 0 positions).  After every step the draft logits of the LAST
    draft pass, the verify logits of the last accepted row, the accepted tokens and kv_len are compared with the
    oracle.  A token may differ only where the oracle's own margin (draft or verify) is below 1e-3 (Q23); that
    ends the comparison for the prompt, and further prompts run until 8 spec steps have been compared."""
    if shape == "c3":
        cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True)
    else:
        cfg = replace(S.config_small_bf16(gates=(1,), accel_end_layer=1, lm_head_adapter=True), name="S-gemma", d_model=384,
                      n_heads=3, head_dim=128, accel_heads=(0,), vocab=19997)
    W = S.gen_weights(cfg)
    compared = 0
    for prompt_seed in range(4):
        eng, orc = M.Engine(cfg, W), Oracle(cfg, W)
        prompt = S.gen_prompt(cfg, 23 + prompt_seed, seed=1000 + prompt_seed)
        fo, fe = orc.prefill(prompt), int(eng.prefill(prompt)[0])
        ok = orc.margin() >= MARGIN
        assert fe == fo or not ok
        for step in range(10):
            if not ok:
                break
            gamma = (2, 4, 6, 1, 3)[step % 5]
            acc_o, _ = orc.spec_step(gamma)
            acc_e, n_e = eng.spec_step(gamma)
            ok = orc.step_margin() >= MARGIN
            got = acc_e[0][:n_e[0]].tolist()
            if got != acc_o:
                assert not ok, (step, got, acc_o, orc.step_margin())
                break
            check_logits(cfg, eng.debug_read(M.DBG_EXIT_LOGITS, 0), orc.exit_logits(0), "draft logits")
            check_logits(cfg, eng.debug_read(M.DBG_LOGITS, gamma), orc.logits(), "verify logits")
            assert eng.get_stats()["kv_len"][0] == orc.kv_len
            compared += 1
        eng.close()
        orc.close()
        if compared >= 8:
            break
    assert compared >= 8, compared


def test_draft_logits_every_draft_position_matches_oracle():
    """The fused draft pass at joff = 0..3: a spec_step(j + 1) on a fresh pair of engines ends with the draft
    pass at joff = j, so DBG_EXIT_LOGITS / orc.exit_logits(0) hold that pass's logits (LM-head adapter on)."""
    cfg = S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True)
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 40)
    for j in range(4):
        eng, orc = M.Engine(cfg, W), Oracle(cfg, W)
        eng.prefill(prompt)
        orc.prefill(prompt)
        acc_o, dr_o = orc.spec_step(j + 1)
        acc_e, n_e = eng.spec_step(j + 1)
        if orc.step_margin() >= MARGIN and acc_e[0][:n_e[0]].tolist() == acc_o:
            check_logits(cfg, eng.debug_read(M.DBG_EXIT_LOGITS, 0), orc.exit_logits(0), "draft logits joff %d" % j)
        eng.close()
        orc.close()


def test_c5_full_size_three_policies_match_oracle():
    """BASELINE configs[4] at FULL size (16 layers, d 2048, 16 x 128 heads, 8 experts x 5632, top-2, 2 slots
    per layer, predictor source p_4 -> layers 4..15), prompt 32, 4 teacher-forced steps under each of the three
    policies: hidden states of both streams, logits, routed and predicted expert indices, router weights and
    the cache counters against the oracle's logical LRU model."""
    cfg = replace(S.config_c5(), max_seq=64)
    eng = M.Engine(cfg)
    W = S.gen_weights(cfg, expert_alloc=eng.pinned_expert_alloc())
    eng.load_weights(W)
    orc = Oracle(cfg, W)
    prompt = S.gen_prompt(cfg, 32)
    for policy in (M.POLICY_FIXED, M.POLICY_LRU, M.POLICY_LRU_AOT):
        eng.set_policy(policy)
        orc.reset()
        orc.set_policy(policy)
        fo, fe = orc.prefill(prompt), int(eng.prefill(prompt)[0])
        assert fe == fo or orc.margin() < MARGIN
        for s in range(4):
            tok_in = orc.pending
            orc.decode_step()
            eng.decode_step(force_tokens=[tok_in])
            assert compare_decode_step(cfg, eng, orc, M) <= 1e-2
            ri = eng.debug_read(M.DBG_ROUTE_IDX).reshape(cfg.n_layers, cfg.top_k).astype(np.int32)
            assert np.array_equal(ri, orc.route_idx()), (policy, s)
            assert np.allclose(eng.debug_read(M.DBG_ROUTE_W).reshape(cfg.n_layers, cfg.top_k), orc.route_w(), atol=2e-3)
            if policy == M.POLICY_LRU_AOT:
                pi = eng.debug_read(M.DBG_PRED_IDX).reshape(cfg.n_layers, cfg.top_k).astype(np.int32)
                po = orc.pred_idx()
                assert np.array_equal(pi[po >= 0], po[po >= 0]), (s, pi, po)
                assert (po[4:] >= 0).all() and (po[:4] == -1).all()
            st, so = eng.get_stats(), orc.stats()
            assert (st["expert_hits"], st["expert_misses"], st["expert_prefetched"], st["expert_on_demand"]) == \
                   (so["expert_hits"], so["expert_misses"], so["prefetched"], so["on_demand"]), (policy, s, st, so)
    eng.close()
    orc.close()


def test_c4_full_width_batch8_passes_match_per_operation_kernels():
    """BASELINE configs[3] at FULL width (d 3072, 32 layers, F 8192, vocabulary 32064) and batch 8, context 1024 to bound
    the time: the batched passes as bench.py times them — 16 dual rows per draft pass and 40 verify rows on
    rows_mma_kernel (rows packed once, K split of all four matrices with second-stage epilogues, adapters, RoPE + KV append
    in the QKV epilogue), tensor-core attention, the draft head on the tensor-core GEMM — against the per-operation
    kernels of the same library (row-major fp32-FMA GEMV, separate RoPE kernel) on the same scripted spec_step: accepted
    tokens, logits of every verify row of sequences 0, 3 and 7, the K/V rows the step appended.  Both engines prefill
    on the fast path; the second switches to the per-operation kernels for the step."""
    B, P, gamma, alpha = 8, 1024, 4, 0.7
    cfg = replace(S.config_c4(), max_seq=P + 64)
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    prompts = np.stack([S.gen_prompt(cfg, P, seq=q) for q in range(B)])
    scripts = [S.gen_logit_script(cfg, 64, alpha, seq=q) for q in range(B)]
    for e in (a, b):
        e.set_logit_script(np.stack([s[0] for s in scripts]), np.stack([s[1] for s in scripts]), P)
        first = e.prefill(prompts)
        assert [int(t) for t in first] == [int(s[0][0]) for s in scripts]
    b.set_fused(False)
    acc_a, n_a = a.spec_step(gamma)
    acc_b, n_b = b.spec_step(gamma)
    assert n_a.tolist() == n_b.tolist()
    for q in range(B):
        assert acc_a[q][:int(n_a[q])].tolist() == acc_b[q][:int(n_b[q])].tolist()
    for q in (0, 3, 7):
        for j in range(gamma + 1):
            la, lb = a.debug_read(M.DBG_LOGITS, j, q), b.debug_read(M.DBG_LOGITS, j, q)
            err, rel = float(np.max(np.abs(la - lb))), rel_l2(la, lb)
            assert err <= 5e-2 and rel <= 5e-3, (q, j, err, rel)
        T = a.get_stats()["kv_len"][q]
        assert T == b.get_stats()["kv_len"][q] and T > P
        for layer in (0, cfg.n_layers - 1):
            for v in (False, True):
                ka, kb = a.kcache(layer, T, b=q, v=v), b.kcache(layer, T, b=q, v=v)
                assert rel_l2(ka[P:], kb[P:]) <= 1e-2, (q, layer, v, rel_l2(ka[P:], kb[P:]))
    a.close()
    b.close()


def test_c4_reduced_width_full_length_batch8():
    """BASELINE configs[3] at FULL length and batch (B = 8 sequences x 4096-token KV, spec_step(4), per-sequence
    scripts so that kv_len diverges) on a reduced-width model (8 heads x 96, 2 layers): the batched per-operation
    path with long-context split-K attention (32 splits of 128 positions), 40 verify rows.  Sequences 0 and 7 are
    followed by their own oracle (accepted tokens, kv_len, K/V after rollback, verify logits); every sequence's
    accepted lengths and kv_len are checked against the closed form of the script (I10)."""
    B, P, gamma, alpha = 8, 4096, 4, 0.7
    cfg = replace(S.config_small_bf16(), name="C4-narrow", n_layers=2, d_model=768, n_heads=8, d_ff=1024, vocab=2048,
                  accel_heads=(0, 1), gates=(1,), accel_end_layer=1, lm_head_adapter=True, max_batch=B,
                  max_seq=P + 64, seed=0x4D325232 + 22)
    W = S.gen_weights(cfg)
    eng = M.Engine(cfg, W)
    prompts = np.stack([S.gen_prompt(cfg, P, seq=b) for b in range(B)])
    scripts = [S.gen_logit_script(cfg, 64, alpha, seq=b) for b in range(B)]
    eng.set_logit_script(np.stack([s[0] for s in scripts]), np.stack([s[1] for s in scripts]), P)
    followed = {0: Oracle(cfg, W), 7: Oracle(cfg, W)}
    first = eng.prefill(prompts)
    for b, o in followed.items():
        o.set_logit_script(scripts[b][0], scripts[b][1], P)
        assert int(first[b]) == o.prefill(prompts[b]) == scripts[b][0][0]
        check_logits(cfg, eng.debug_read(M.DBG_LOGITS, (P - 1) % 8, b), o.logits(), "prefill logits seq %d" % b)
    pos = [P] * B
    for step in range(5):
        acc, n = eng.spec_step(gamma)
        kv = eng.get_stats()["kv_len"]
        for b in range(B):
            f, g = scripts[b]
            a = 0
            while a < gamma and g[pos[b] + 1 + a - P] == f[pos[b] + 1 + a - P]:
                a += 1
            assert int(n[b]) == a + 1, (step, b, n[b], a)
            assert acc[b][:a + 1].tolist() == f[pos[b] + 1 - P: pos[b] + 2 + a - P].tolist()
            pos[b] += a + 1
            assert kv[b] == pos[b]
        for b, o in followed.items():
            ao, _ = o.spec_step(gamma)
            assert acc[b][:n[b]].tolist() == ao and o.kv_len == pos[b]
            check_logits(cfg, eng.debug_read(M.DBG_LOGITS, gamma, b), o.logits(), "verify logits seq %d" % b)
    assert len(set(pos)) > 1, "scripts should make kv_len diverge"
    for b, o in followed.items():
        T = o.kv_len
        for i in range(cfg.n_layers):
            assert rel_l2(eng.kcache(i, T, b=b)[P - 8:], o.kcache(i)[P - 8:T]) <= 1e-2
            assert rel_l2(eng.kcache(i, T, b=b, v=True), o.vcache(i)[:T]) <= 1e-2
        o.close()
    eng.close()


# ------------------------------------------------------------------ f-1: top-k token-subset accelerated attention
TOPK_SEL_MARGIN = 1e-4   # a step is compared only where the oracle's k-th and (k+1)-th slow scores are this far apart


@pytest.mark.parametrize("dtype,k,P", [(S.FP32, 8, 40), (S.BF16, 16, 90)])
def test_topk_token_subset_accelerated_attention_matches_oracle(dtype, k, P):
    """PAPER.md L158, footnote 4 L170: with accel_topk_tokens = k the accelerated stream of a head in S
    attends only the k cached positions with the largest slow-stream scores plus its own key (`accel_topk_attn_kernel`,
    per-operation path).  Every h_i, p_i, the logits and the tokens against the oracle under teacher forcing, on fp32
    (rel-L2 1e-4) and bf16 storage; the selection is an integer decision taken from fp32 scores on both sides, so a step
    whose selection margin in the oracle is below 1e-4 is re-synchronised but not compared (Q21)."""
    base = S.config_c1() if dtype == S.FP32 else S.config_small_bf16()
    cfg = replace(base, accel_topk_tokens=k, max_seq=max(base.max_seq, P + 16))
    W = S.gen_weights(cfg)
    eng, orc = M.Engine(cfg, W), Oracle(cfg, W)
    dense = Oracle(replace(cfg, accel_topk_tokens=0), W)
    prompt = S.gen_prompt(cfg, P)
    fe, fo = int(eng.prefill(prompt)[0]), orc.prefill(prompt)
    dense.prefill(prompt)
    assert fe == fo or orc.margin() < MARGIN
    compared, restricted = 0, False
    for s in range(8):
        tok_in = orc.pending
        to, _ = orc.decode_step()
        dense.decode_step(force_token=tok_in)
        te = eng.decode_step(force_tokens=[tok_in])
        assert eng.get_stats()["kv_len"][0] == orc.kv_len
        if orc.topk_margin() < TOPK_SEL_MARGIN:
            continue
        compare_decode_step(cfg, eng, orc, M)
        assert int(te[0]) == to or orc.margin() < MARGIN
        restricted |= rel_l2(orc.trace_p()[1], dense.trace_p()[1]) > 1e-6
        compared += 1
    assert compared >= 5 and restricted          # the restriction is active and most steps are comparable
    eng.close()


def test_topk_token_subset_selfspec_is_lossless_on_gpu():
    """Self-speculation with the top-k accelerated attention: drafts come from the restricted accelerated stream, the
    verify pass is the unchanged slow stream, so the emitted stream equals plain greedy decoding token for token (I7)."""
    cfg = replace(S.config_small_bf16(gates=(2,), accel_end_layer=2, lm_head_adapter=True), accel_topk_tokens=16)
    W = S.gen_weights(cfg)
    a, b = M.Engine(cfg, W), M.Engine(cfg, W)
    orc = Oracle(cfg, W)
    prompt = S.gen_prompt(cfg, 50)
    a.prefill(prompt); b.prefill(prompt); orc.prefill(prompt)
    spec, plain, n_ok = [], [], 0
    for _ in range(6):
        acc, n = a.spec_step(3)
        ao, _ = orc.spec_step(3)
        if not (orc.step_margin() >= MARGIN and orc.topk_margin() >= TOPK_SEL_MARGIN):
            break                                 # a near-tie: nothing after it is comparable token for token
        assert acc[0][:n[0]].tolist() == ao
        spec += acc[0][:n[0]].tolist()
        n_ok += 1
    while len(plain) < len(spec):
        plain.append(int(b.decode_step()[0]))
    assert spec == plain[:len(spec)] and n_ok >= 3
    a.close(); b.close()


# ------------------------------------------------------------------ f-3: ARLA mechanics
@pytest.mark.parametrize("which", ["c1-fp32", "small-bf16-fused", "small-bf16-per-op"])
def test_arla_exit_scores_match_oracle(which):
    """the exit score of every gate, sigma(w_o . softmax(q K^T / sqrt(d^s)) V + b)
    over the latent projections (d^s = 64, footnote 2) of the interval's accelerated residuals, computed by `arla_kernel`
    from the traces of the decode step (fused kernel or per-operation kernels), against the oracle under teacher forcing."""
    if which == "c1-fp32":
        cfg, tol = replace(S.config_c1(), arla_dim=64), 2e-5
    else:
        cfg, tol = S.config_small_bf16(arla_dim=64), 2e-3
    W = S.gen_weights(cfg)
    eng, orc = M.Engine(cfg, W), Oracle(cfg, W)
    if which == "small-bf16-per-op":
        eng.set_fused(False)
    prompt = S.gen_prompt(cfg, 21)
    eng.prefill(prompt); orc.prefill(prompt)
    seen = []
    for s in range(5):
        tok_in = orc.pending
        orc.decode_step()
        eng.decode_step(force_tokens=[tok_in])
        got, want = eng.debug_read(M.DBG_EXIT_SCORE), orc.exit_scores()
        assert got.shape == want.shape == (len(cfg.gates),)
        assert np.max(np.abs(got - want)) <= tol, (s, got, want)
        seen.append(want.copy())
    assert np.ptp(np.stack(seen)) > 1e-4          # the scores depend on the token
    eng.close()
