"""Pins for the CPU oracle.  All CPU-only (`-m "not gpu"`).

The paper prints no worked numeric example (every number is inside a figure image), so the
oracle is pinned by: a special case that reduces to torch library routines (I1), brute
force on tiny inputs (I5, I15), closed forms (I10, I12, I16, I17) and invariants the paper
fixes (I2-I4, I6-I9, I13, I14).  Each test names the passage it follows.
"""
from dataclasses import replace

import numpy as np
import pytest

import m2r2_synth as S
from oracle import Oracle
from tests.refs import (np_accel_layer, np_accel_layer_moe, np_moe_slow_layer, np_rms, np_rope, np_route, rel_l2,
                        torch_decoder)


def tiny(**kw):
    base = replace(S.config_c1(), n_layers=3, d_model=64, n_heads=4, head_dim=16, d_ff=96,
                   vocab=211, max_seq=64, accel_heads=(1, 3), gates=(2,), accel_end_layer=3,
                   adapter_rank=4)
    return replace(base, **kw)


def run_plain(cfg, W, prompt, n_new, **okw):
    o = Oracle(cfg, W)
    toks = [o.prefill(prompt)]
    for _ in range(n_new - 1):
        toks.append(o.decode_step()[0])
    return toks, o


# ---------------------------------------------------------------- I1
@pytest.mark.parametrize("dtype", [S.FP32, S.BF16])
def test_I1_slow_stream_is_textbook_prenorm_decoder(dtype):
    """PAPER.md Eq. 1 (L47-50) + norms (L60): with the accelerated stream off the oracle
    equals a pre-norm decoder built from torch ops over the full sequence (BASELINE inv. 1)."""
    cfg = replace(S.config_c1(), dtype=dtype, accel_enabled=False, gates=(), accel_end_layer=0)
    W = S.gen_weights(cfg)
    seq = S.gen_prompt(cfg, 24)
    hid, logits = torch_decoder(cfg, W, seq)
    P = 16
    o = Oracle(cfg, W)
    o.prefill(seq[:P])
    tol = 1e-5 if dtype == S.FP32 else 2e-3   # bf16: K/V rounding boundaries can flip
    assert rel_l2(o.logits(), logits[P - 1]) < tol
    for t in range(P, len(seq)):
        o.decode_step(force_token=int(seq[t]))
        H = o.trace_h()
        for i in range(cfg.n_layers + 1):
            assert rel_l2(H[i], hid[i, t]) < tol, (t, i)
        assert rel_l2(o.logits(), logits[t]) < tol
        if dtype == S.FP32:
            assert int(np.argmax(logits[t])) == o.pending


def test_I1_c1_prefill_matches_textbook_at_every_prefix():
    cfg = replace(S.config_c1(), accel_enabled=False, gates=(), accel_end_layer=0)
    W = S.gen_weights(cfg)
    seq = S.gen_prompt(cfg, 12)
    _, logits = torch_decoder(cfg, W, seq)
    for P in (1, 2, 7, 12):
        o = Oracle(cfg, W)
        tok = o.prefill(seq[:P])
        assert rel_l2(o.logits(), logits[P - 1]) < 1e-5
        assert tok == int(np.argmax(logits[P - 1]))


# ---------------------------------------------------------------- I2
def test_I2_slow_stream_never_reads_accelerated_stream():
    """PAPER.md L74 (base model untouched; adapters are parallel): h and tokens bit-identical
    with the accelerated stream on or off."""
    cfg_on = tiny()
    cfg_off = replace(cfg_on, accel_enabled=False)
    W = S.gen_weights(cfg_on)
    prompt = S.gen_prompt(cfg_on, 9)
    a, oa = run_plain(cfg_on, W, prompt, 12)
    b, ob = run_plain(cfg_off, W, prompt, 12)
    assert a == b
    assert np.array_equal(oa.trace_h(), ob.trace_h())
    assert np.array_equal(oa.logits(), ob.logits())
    for i in range(cfg_on.n_layers):
        assert np.array_equal(oa.kcache(i)[:oa.kv_len], ob.kcache(i)[:ob.kv_len])


# ---------------------------------------------------------------- I3
def test_I3_zero_adapters_all_heads_gives_p_equal_h():
    """Induction on Eq. 2 (L70) with L76: if B=0 and S = all heads then p_i == h_i (k^_t = k_t
    up to cache rounding, so fp32 here), exit tokens at E=N equal final tokens, and self-spec
    from E=N accepts every draft."""
    cfg = tiny(accel_heads=(0, 1, 2, 3), gates=(3,), accel_end_layer=3)
    W = S.gen_weights(cfg)
    S.zero_adapters(cfg, W)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 7))
    for _ in range(5):
        tok, ex = o.decode_step()
        assert rel_l2(o.trace_p(), o.trace_h()) < 1e-6
        assert ex[0] == tok
    for g in (1, 3, 5):
        acc, dr = o.spec_step(g)
        assert len(acc) == g + 1 and acc[:g] == dr


# ---------------------------------------------------------------- I4
def test_I4_gate_reinitialises_p_from_h():
    """PAPER.md L82 / L101: p_{E_j} <- h_{E_j} (identity) at pass start and at each gate."""
    cfg = tiny(gates=(2,), accel_end_layer=3)
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 6))
    o.decode_step()
    H, P = o.trace_h(), o.trace_p()
    t = o.kv_len - 1
    assert np.array_equal(P[0], H[0])                      # p_0 = h_0
    assert not np.array_equal(P[2], H[2])                  # p_2 (pre-reset) differs from h_2
    # layer 2 of the accelerated stream must have started from h_2, not from p_2
    assert np.array_equal(o.accel_layer(2, H[2], t), P[3])
    assert not np.array_equal(o.accel_layer(2, P[2], t), P[3])
    # and layers 0,1 chain from p_0 = h_0
    p1 = o.accel_layer(0, H[0], t)
    assert np.array_equal(p1, P[1])
    assert np.array_equal(o.accel_layer(1, p1, t), P[2])


# ---------------------------------------------------------------- I5
@pytest.mark.parametrize("dtype", [S.FP32, S.BF16])
def test_I5_accelerated_attention_bruteforce(dtype):
    """A^ = MHA(p_t, h_{<t} (+) p_t, h_{<t} (+) p_t) — brute force with the
    explicit (t+1)-row key/value matrix [K[0..t-1]; k^_t]; slow K[t]/V[t] must be invisible."""
    cfg = tiny(dtype=dtype)
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 8))
    o.decode_step()
    H, P = o.trace_h(), o.trace_p()
    t = o.kv_len - 1
    for i in (0, 1):
        want = np_accel_layer(cfg, W["layers"][i], P[i], t, o.kcache(i), o.vcache(i))
        assert rel_l2(P[i + 1], want) < 2e-6, i
    # perturbing the slow stream's own K[t], V[t] leaves the accelerated output unchanged ...
    base = o.accel_layer(1, P[1], t)
    o.kcache(1)[t] += 3.0
    o.vcache(1)[t] -= 5.0
    assert np.array_equal(o.accel_layer(1, P[1], t), base)
    # ... while perturbing any cached position < t changes it
    o.vcache(1)[t - 1] += 1.0
    assert not np.array_equal(o.accel_layer(1, P[1], t), base)
    # t = 0: the only key is the token's own k^_0 -> softmax weight 1 -> o^ = v^_0
    o0 = Oracle(cfg, W)
    o0.prefill(S.gen_prompt(cfg, 1))
    p = H[0]
    want0 = np_accel_layer(cfg, W["layers"][0], p, 0, o0.kcache(0), o0.vcache(0))
    assert rel_l2(o0.accel_layer(0, p, 0), want0) < 2e-6


# ---------------------------------------------------------------- I24
@pytest.mark.parametrize("dtype", [S.FP32, S.BF16])
def test_I24_topk_token_subset_accelerated_attention(dtype):
    """PAPER.md L158, footnote 4 L170 (Q21): per head, p attends only the k cached positions with the largest
    slow-stream attention coefficients (same head, same token) plus its own key.
    (a) brute force in numpy float64 from the traces, the slow cache and the weights (selection from the SLOW query);
    (b) k >= t is the dense accelerated attention, bit for bit; the slow stream never changes;
    (c) with k < t the result differs from the dense one (the restriction is real) and perturbing a NON-selected cached
        position's V leaves the accelerated output unchanged while a selected one changes it."""
    k = 6
    cfg = tiny(dtype=dtype, accel_topk_tokens=k)
    dense = tiny(dtype=dtype)
    W = S.gen_weights(cfg)
    o, od = Oracle(cfg, W), Oracle(dense, W)
    prompt = S.gen_prompt(cfg, 19)
    assert o.prefill(prompt) == od.prefill(prompt)
    for step in range(3):
        tok = od.pending
        o.decode_step(force_token=tok)
        od.decode_step(force_token=tok)
        H, P = o.trace_h(), o.trace_p()
        assert np.array_equal(H, od.trace_h())                       # the slow stream is untouched
        t = o.kv_len - 1
        assert t > k and np.isfinite(o.topk_margin()) and o.topk_margin() > 0
        differs = False
        for i in range(cfg.accel_end_layer):
            gated = i in cfg.gates
            p_in = H[i] if (i == 0 or gated) else P[i]
            want = np_accel_layer(cfg, W["layers"][i], p_in, t, o.kcache(i), o.vcache(i), h=H[i], topk=k)
            assert rel_l2(P[i + 1], want) < 2e-6, (step, i)
            differs |= rel_l2(P[i + 1], od.trace_p()[i + 1]) > 1e-6
        assert differs
    # (b) k >= t: identical to dense
    big = Oracle(tiny(dtype=dtype, accel_topk_tokens=64), W)
    od2 = Oracle(dense, W)
    big.prefill(prompt); od2.prefill(prompt)
    big.decode_step(); od2.decode_step()
    assert np.array_equal(big.trace_p(), od2.trace_p()) and not np.isfinite(big.topk_margin())
    # (c) selection is what restricts: layer 0, head S[0]
    t = o.kv_len - 1
    H = o.trace_h()
    a, dh = cfg.accel_heads[0], cfg.head_dim
    from tests.refs import np_rms, np_rope
    f = lambda key: S.as_f32(cfg, W["layers"][0][key]).astype(np.float64)
    qs = np_rope(cfg, (f("wq") @ np_rms(cfg, H[0], f("g1"))).astype(np.float32), t)[a * dh:(a + 1) * dh]
    ss = o.kcache(0)[:t, a * dh:(a + 1) * dh].astype(np.float64) @ qs
    order = sorted(range(t), key=lambda u: (-ss[u], u))
    chosen, dropped = order[0], order[-1]
    o.slow_layer(0, H[0], t)             # re-runs slow layer 0 of this token: the oracle now holds ITS slow query again
    base = o.accel_layer(0, H[0], t)
    o.vcache(0)[dropped, a * dh:(a + 1) * dh] += 7.0
    assert np.array_equal(o.accel_layer(0, H[0], t), base)
    o.vcache(0)[chosen, a * dh:(a + 1) * dh] += 7.0
    assert not np.array_equal(o.accel_layer(0, H[0], t), base)


# ---------------------------------------------------------------- I25
@pytest.mark.parametrize("gates", [(2,), (1, 3)])
def test_I25_arla_exit_scores_bruteforce(gates):
    """PAPER.md L105-117, Fig. 4a (Q26): the exit score of gate E_j = sigma(w_o . softmax(q K^T / sqrt(d^s)) V + b)
    with K, V the latent projections of the interval's residuals (the state p was re-initialised from, then every p_i up
    to the one before the reset) and q the projection of the LAST one.  (a) numpy float64 brute force from the traces;
    (b) W_v = 0 => sigma(b); (c) W_q = 0 => uniform attention => the value is the mean of the interval's V."""
    ds = 8
    cfg = tiny(arla_dim=ds, gates=gates)
    W = S.gen_weights(cfg)
    d = cfg.d_model

    def brute(Wm, H, P):
        A = S.as_f32(cfg, Wm["arla"]).astype(np.float64).reshape(len(gates), 3 * ds + 1, d)
        out = []
        for j, hi in enumerate(gates):
            lo = gates[j - 1] if j else 0
            Z = np.stack([H[lo]] + [P[i] for i in range(lo + 1, hi + 1)]).astype(np.float64)
            Wq, Wk, Wv, wo, b = A[j, :ds], A[j, ds:2 * ds], A[j, 2 * ds:3 * ds], A[j, 3 * ds, :ds], A[j, 3 * ds, ds]
            q, K, V = Wq @ Z[-1], Z @ Wk.T, Z @ Wv.T
            sc = K @ q / np.sqrt(ds)
            a = np.exp(sc - sc.max()); a /= a.sum()
            out.append(1.0 / (1.0 + np.exp(-(wo @ (a @ V) + b))))
        return np.array(out)

    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 7))
    for _ in range(3):
        o.decode_step()
        got = o.exit_scores()
        want = brute(W, o.trace_h(), o.trace_p())
        assert np.allclose(got, want, atol=2e-6), (got, want)
        assert np.all((got > 0) & (got < 1)) and np.ptp(got) > 0 or len(gates) == 1
    # (b), (c): edited copies of the router
    A = W["arla"].reshape(len(gates), 3 * ds + 1, d)
    Wb = dict(W); Ab = A.copy(); Ab[:, 2 * ds:3 * ds] = 0; Wb["arla"] = np.ascontiguousarray(Ab.reshape(-1, d))
    ob = Oracle(cfg, Wb); ob.prefill(S.gen_prompt(cfg, 7)); ob.decode_step()
    bias = S.as_f32(cfg, W["arla"]).reshape(len(gates), 3 * ds + 1, d)[:, 3 * ds, ds].astype(np.float64)
    assert np.allclose(ob.exit_scores(), 1.0 / (1.0 + np.exp(-bias)), atol=1e-6)
    Wc = dict(W); Ac = A.copy(); Ac[:, :ds] = 0; Wc["arla"] = np.ascontiguousarray(Ac.reshape(-1, d))
    oc = Oracle(cfg, Wc); oc.prefill(S.gen_prompt(cfg, 7)); oc.decode_step()
    Af = S.as_f32(cfg, W["arla"]).astype(np.float64).reshape(len(gates), 3 * ds + 1, d)
    H, P = oc.trace_h(), oc.trace_p()
    for j, hi in enumerate(gates):
        lo = gates[j - 1] if j else 0
        Z = np.stack([H[lo]] + [P[i] for i in range(lo + 1, hi + 1)]).astype(np.float64)
        v = (Z @ Af[j, 2 * ds:3 * ds].T).mean(axis=0)
        want = 1.0 / (1.0 + np.exp(-(Af[j, 3 * ds, :ds] @ v + Af[j, 3 * ds, ds])))
        assert abs(oc.exit_scores()[j] - want) < 2e-6


# ---------------------------------------------------------------- I6
def test_I6_incremental_equals_recompute():
    """KV-cache indexing: prefill(P) + q decode steps == prefill(P+q) at every position."""
    cfg = tiny()
    W = S.gen_weights(cfg)
    seq = S.gen_prompt(cfg, 14)
    o = Oracle(cfg, W)
    o.prefill(seq[:5])
    for t in range(5, 14):
        o.decode_step(force_token=int(seq[t]))
        full = Oracle(cfg, W)
        full.prefill(seq[:t + 1])
        assert np.array_equal(o.logits(), full.logits())
        for i in range(cfg.n_layers):
            assert np.array_equal(o.kcache(i)[:t + 1], full.kcache(i)[:t + 1])
            assert np.array_equal(o.vcache(i)[:t + 1], full.vcache(i)[:t + 1])


# ---------------------------------------------------------------- I7, I8, I9
@pytest.mark.parametrize("E", [1, 2, 3])
@pytest.mark.parametrize("gamma", [0, 1, 2, 3, 4, 5, 6])
def test_I7_selfspec_is_lossless(E, gamma):
    """speculative decoding does not change the greedy output."""
    cfg = tiny(gates=(E,), accel_end_layer=E)
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 6)
    ref, _ = run_plain(cfg, W, prompt, 24)
    o = Oracle(cfg, W)
    out = [o.prefill(prompt)]
    n = len(prompt)
    while len(out) < 24:
        acc, dr = o.spec_step(gamma)
        assert 1 <= len(acc) <= gamma + 1
        out += acc
        n += len(acc)
        assert o.kv_len == n and o.pending == out[-1]
    assert out[:24] == ref


def test_I8_rollback_leaves_cache_equal_to_plain_decode():
    """BASELINE inv. 3: after rejected drafts and rollback, K/V[0..kv_len) equal plain
    decode's, dead positions are never read (NaN poison), and plain decode continues."""
    cfg = tiny(gates=(1,), accel_end_layer=1)   # E=1 -> poor drafts -> many rejections
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 6)
    ref, oref = run_plain(cfg, W, prompt, 30)
    o = Oracle(cfg, W)
    out = [o.prefill(prompt)]
    rejected = 0
    while len(out) < 14:
        acc, dr = o.spec_step(4)
        rejected += 4 - (len(acc) - 1)
        out += acc
        for i in range(cfg.n_layers):     # poison everything beyond kv_len
            o.kcache(i)[o.kv_len:] = np.nan
            o.vcache(i)[o.kv_len:] = np.nan
    assert rejected > 0
    L = o.kv_len
    # the plain run has decoded further; its first L positions must be identical
    for i in range(cfg.n_layers):
        assert np.array_equal(o.kcache(i)[:L], oref.kcache(i)[:L])
        assert np.array_equal(o.vcache(i)[:L], oref.vcache(i)[:L])
    while len(out) < 30:
        out.append(o.decode_step()[0])
    assert out[:30] == ref


def test_I9_spec_step_zero_equals_decode_step():
    cfg = tiny()
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 5)
    a, b = Oracle(cfg, W), Oracle(cfg, W)
    a.prefill(prompt)
    b.prefill(prompt)
    for _ in range(6):
        ta, _ = a.decode_step()
        acc, _ = b.spec_step(0)
        assert acc == [ta] and a.kv_len == b.kv_len
        assert np.array_equal(a.logits(), b.logits())
        for i in range(cfg.n_layers):
            assert np.array_equal(a.kcache(i)[:a.kv_len], b.kcache(i)[:b.kv_len])


# ---------------------------------------------------------------- I10
@pytest.mark.parametrize("alpha", [0.5, 0.9])
@pytest.mark.parametrize("gamma", [2, 4, 6])
def test_I10_closed_form_acceptance_under_logit_script(alpha, gamma):
    """SURVEY §8(d) logit script: plain greedy output is exactly f_s, and
    n_accepted - 1 = min(gamma, first j with g_{n+1+j} != f_{n+1+j}) — from the seed alone."""
    cfg = tiny(gates=(2,), accel_end_layer=2)
    W = S.gen_weights(cfg)
    P = 5
    prompt = S.gen_prompt(cfg, P)
    f, g = S.gen_logit_script(cfg, 64, alpha)
    o = Oracle(cfg, W)
    o.set_logit_script(f, g, first_pos=P)
    first = o.prefill(prompt)
    assert first == f[0]                      # token at position P is f_P
    n, emitted = P, [first]
    while n + gamma + 1 < P + 56:
        acc, dr = o.spec_step(gamma)
        # drafts d_j predict position n+1+j; verifier tokens t_j predict the same positions
        want_a = 0
        while want_a < gamma and g[n + 1 + want_a - P] == f[n + 1 + want_a - P]:
            want_a += 1
        # drafted tokens follow the script as long as they were fed script-consistent inputs
        assert len(acc) - 1 == want_a, (n, acc, dr)
        assert acc == [int(x) for x in f[n + 1 - P:n + 1 - P + want_a + 1]]
        n += len(acc)
        emitted += acc
        assert o.kv_len == n
    assert emitted == [int(x) for x in f[:len(emitted)]]
    st = o.stats()
    assert st["emitted"] == len(emitted) - 1 and st["drafted"] == st["steps"] * gamma


# ---------------------------------------------------------------- I12
def test_I12_rope_convention_and_relativity():
    cfg = tiny(head_dim=16)
    o = Oracle(cfg, S.gen_weights(cfg))
    rng = np.random.default_rng(0)
    q = rng.standard_normal(16).astype(np.float32)
    k = rng.standard_normal(16).astype(np.float32)
    assert np.array_equal(o.rope(q, 0), q)                          # rope(v, 0) = v
    for j in (0, 3, 7):                                             # closed form on unit vectors
        e = np.zeros(16, np.float32)
        e[j] = 1
        ang = 5 * cfg.rope_theta ** (-2.0 * j / 16)
        r = o.rope(e, 5)
        want = np.zeros(16)
        want[j], want[j + 8] = np.cos(ang), np.sin(ang)
        assert np.allclose(r, want, atol=1e-7)
    assert np.allclose(o.rope(q, 9), np_rope(cfg, q, 9), atol=1e-6)
    for (t, u, dl) in [(3, 1, 10), (17, 17, 4), (30, 2, 25)]:       # relativity
        a = float(np.dot(o.rope(q, t).astype(np.float64), o.rope(k, u)))
        b = float(np.dot(o.rope(q, t + dl).astype(np.float64), o.rope(k, u + dl)))
        assert abs(a - b) < 1e-5


# ---------------------------------------------------------------- I13
def test_I13_argmax_and_topk_ties_and_router_weights():
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    assert o.argmax(np.array([1, 5, 5, 2], np.float32)) == 1        # lowest index wins
    assert o.argmax(np.array([7, 7, 7], np.float32)) == 0
    d, ne = cfg.d_model, cfg.n_experts
    Wr = np.zeros((ne, d), dtype=np.uint16)                         # all logits equal (0)
    idx, w = o.route(Wr, np.ones(d, np.float32))
    assert idx.tolist() == [0, 1] and np.allclose(w, [0.5, 0.5])
    # distinct indices, weights sum to one (renormalised over the top-2), match a dense softmax
    y = np.random.default_rng(1).standard_normal(d).astype(np.float32)
    R = W["layers"][0]["router"]
    idx, w = o.route(R, y)
    logits = S.as_f32(cfg, R).astype(np.float64) @ y
    pr = np.exp(logits - logits.max())
    pr /= pr.sum()
    order = np.argsort(-logits, kind="stable")[:2]
    assert idx.tolist() == order.tolist() and idx[0] != idx[1]
    assert abs(w.sum() - 1) < 1e-6
    assert np.allclose(w, pr[order] / pr[order].sum(), atol=1e-6)
    o2 = Oracle(replace(cfg, renorm_topk=False), W)
    _, w2 = o2.route(R, y)
    assert np.allclose(w2, pr[order], atol=1e-6)


# ---------------------------------------------------------------- I14
def test_I14_single_expert_moe_equals_dense_and_policy_independence():
    dense = tiny(accel_enabled=False, gates=(), accel_end_layer=0)
    moe = replace(dense, n_experts=1, top_k=1, d_ff_expert=dense.d_ff, d_ff=0, cache_slots=1)
    Wd = S.gen_weights(dense)
    Wm = {k: v for k, v in Wd.items() if k != "layers"}
    Wm["layers"] = []
    for L in Wd["layers"]:
        M = {k: L[k] for k in ("g1", "g2", "wq", "wk", "wv", "wo")}
        M["router"] = np.zeros((1, dense.d_model), np.float32)
        M["experts"] = [{"ewg": L["wgate"], "ewu": L["wup"], "ewd": L["wdown"]}]
        Wm["layers"].append(M)
    prompt = S.gen_prompt(dense, 6)
    a, oa = run_plain(dense, Wd, prompt, 8)
    b, ob = run_plain(moe, Wm, prompt, 8)
    assert a == b
    assert rel_l2(ob.trace_h(), oa.trace_h()) < 1e-6
    # numeric output independent of cache size / policy (only counters change)
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 5)
    outs = []
    for policy, slots in [(0, 2), (1, 2), (2, 2), (2, 5), (1, 8)]:
        o = Oracle(replace(cfg, cache_slots=slots), W)
        o.set_policy(policy)
        toks = [o.prefill(prompt)] + [o.decode_step()[0] for _ in range(6)]
        outs.append((toks, o.trace_h()))
    for toks, H in outs[1:]:
        assert toks == outs[0][0] and np.array_equal(H, outs[0][1])


# ---------------------------------------------------------------- I15
def _lru_sim(C, events, policy):
    """Brute-force per-layer LRU: list ordered by last-use time."""
    cache = {}   # expert -> last-use stamp
    for s in range(C):
        cache[s] = -s
    stamp, hits, misses, pref = 1, 0, 0, 0
    for kind, idx in events:
        if kind == "pred" and policy < 2:
            continue
        for e in idx:
            if e in cache:
                if kind == "use":
                    hits += 1
            else:
                if kind == "use":
                    misses += 1
                else:
                    pref += 1
                victims = [x for x in cache if x not in idx]
                victim = min(victims, key=lambda x: cache[x])
                del cache[victim]
            cache[e] = stamp
            stamp += 1
    return hits, misses, pref, sorted(cache, key=lambda x: -cache[x])


@pytest.mark.parametrize("policy", [1, 2, 3, 4])
@pytest.mark.parametrize("C", [2, 3, 5])
def test_I15_lru_model_vs_bruteforce(policy, C):
    """PAPER.md L139/L242 (LRU replaced by speculated experts), Fig. 5 L121 (only
    mis-speculated experts load lazily): counters vs a brute-force simulation."""
    cfg = S.config_small_moe(cache_slots=C)
    o = Oracle(cfg, S.gen_weights(cfg))
    o.set_policy(policy)
    rng = np.random.default_rng(C * 10 + policy)
    events = []
    for _ in range(200):
        kind = "pred" if rng.random() < 0.4 else "use"
        a = int(rng.integers(cfg.n_experts))
        b = int((a + 1 + rng.integers(cfg.n_experts - 1)) % cfg.n_experts)
        events.append((kind, [a, b]))
        (o.lru_predict if kind == "pred" else o.lru_use)(3, [a, b])
    hits, misses, pref, order = _lru_sim(C, events, policy)
    st = o.stats()
    assert (st["expert_hits"], st["expert_misses"], st["prefetched"]) == (hits, misses, pref)
    assert st["on_demand"] == st["expert_misses"]
    assert st["expert_hits"] + st["expert_misses"] == 2 * sum(1 for k, _ in events if k == "use")
    assert o.lru()[3].tolist() == order


def test_I15_end_to_end_counters_with_router_script():
    """With a perfect predictor (pi=1) every targeted layer has zero misses; hits+misses =
    top_k * N * steps; with C = n_e nothing is ever loaded after warm-up."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    P, steps = 4, 12
    actual, pred = S.gen_router_script(cfg, steps, rho=0.25, pi=1.0)
    o = Oracle(cfg, W)
    o.set_policy(2)
    o.set_router_script(actual, pred, first_pos=P)
    o.prefill(S.gen_prompt(cfg, P))
    targeted = sorted({L for lo, hi in cfg.aot_targets for L in range(lo, hi)})
    assert targeted == [2, 3, 4, 5]
    miss_layers_before = o.stats()["expert_misses"]
    assert miss_layers_before == 0            # prefill does not touch the cache model
    for s in range(steps):
        o.decode_step()
        assert np.array_equal(o.route_idx(), actual[s])
        assert np.array_equal(o.pred_idx()[2:], pred[s][2:])
    st = o.stats()
    assert st["expert_hits"] + st["expert_misses"] == cfg.top_k * cfg.n_layers * steps
    # misses can only come from the untargeted layers 0 and 1
    o2 = Oracle(cfg, W)
    o2.set_policy(1)
    o2.set_router_script(actual, pred, first_pos=P)
    o2.prefill(S.gen_prompt(cfg, P))
    for s in range(steps):
        o2.decode_step()
    per_layer_lru_misses = 0
    for L in (0, 1):
        h, m, _, _ = _lru_sim(cfg.cache_slots, [("use", actual[s][L].tolist()) for s in range(steps)], 1)
        per_layer_lru_misses += m
    assert st["expert_misses"] == per_layer_lru_misses
    assert o2.stats()["expert_misses"] >= st["expert_misses"]
    big = Oracle(replace(cfg, cache_slots=cfg.n_experts), W)
    big.set_policy(1)
    big.prefill(S.gen_prompt(cfg, P))
    for s in range(steps):
        big.decode_step()
    assert big.stats()["expert_misses"] == 0


# ---------------------------------------------------------------- I16, I17
def test_I16_aot_targets_rate2_is_2i_plus_2_and_3():
    """with a 2x stream, layer i identifies experts of 2i+2, 2i+3."""
    N = 16
    tg = S.aot_targets_for_rate(N, 2)
    with open(__file__.replace("test_oracle_pins.py", "golden/aot_rate2_targets.txt")) as fh:
        rows = [tuple(int(x) for x in ln.split()) for ln in fh if ln.strip() and ln[0] != "#"]
    for i, a, b in rows:
        assert list(range(*tg[i])) == [x for x in (a, b) if x < N], i
    for i in range(N):
        assert list(range(*tg[i])) == [x for x in (2 * i + 2, 2 * i + 3) if x < N]
    # and the oracle predicts exactly for those targets
    cfg = S.config_small_moe()
    o = Oracle(cfg, S.gen_weights(cfg))
    o.set_policy(2)
    o.prefill(S.gen_prompt(cfg, 3))
    o.decode_step()
    pi = o.pred_idx()
    assert (pi[:2] == -1).all() and (pi[2:] >= 0).all()


def test_I17_equally_spaced_gates_give_rates_Jplus1_to_2():
    """"2-(J+1)x rate"; interval j runs at (N - E_j)/(E_{j+1} - E_j) (Eq. 4)."""
    c = S.config_c2()
    N, g = c.n_layers, (0,) + c.gates
    rates = [(N - g[j]) // (g[j + 1] - g[j]) for j in range(len(c.gates))]
    assert rates == [4, 3, 2]


# ---------------------------------------------------------------- regression fixture
def test_golden_c1_tokens_regression():
    """tests/golden/c1_tokens.txt is written by tests/golden/make_golden.py (oracle only)."""
    cfg = S.config_c1()
    W = S.gen_weights(cfg)
    prompt = S.gen_prompt(cfg, 32)
    toks, _ = run_plain(cfg, W, prompt, 32)
    with open(__file__.replace("test_oracle_pins.py", "golden/c1_tokens.txt")) as fh:
        want = [int(x) for ln in fh if ln.strip() and ln[0] != "#" for x in ln.split()]
    assert toks == want


# ---------------------------------------------------------------- I18-I21: the branches VERDICT r1 found unpinned
# ---------------------------------------------------------------- I22, I23: the comparison strategies of PAPER.md L242
def _spec_mix(counter):
    """the counter-based generator of the random-speculation policy, restated (64-bit wrap-around arithmetic)"""
    M = (1 << 64) - 1
    x = (0x5EC0DE5EED + 0x9E3779B97F4A7C15 * (counter + 1)) & M
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & M
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & M
    return x ^ (x >> 31)


def test_I22_random_speculation_draws_and_counters():
    """Policy 3 (L242: LRU + random pre-loading, Q24): before layer L+1 the top_k experts
    spec_mix((t N + L+1) 256 + draw) mod n_e (duplicates skipped) are pre-loaded.  The oracle's predicted indices
    equal the restated draws, the draws are distinct and roughly uniform, and its counters equal the brute-force LRU
    simulation fed with the (pred, use) event sequence."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    P, steps = 5, 10
    o = Oracle(cfg, W)
    o.set_policy(3)
    o.prefill(S.gen_prompt(cfg, P))
    events = {L: [] for L in range(cfg.n_layers)}
    seen = np.zeros(cfg.n_experts, int)
    for s in range(steps):
        o.decode_step()
        t = P + s
        pred, use = o.pred_idx(), o.route_idx()
        assert pred[0].tolist() == [-1] * cfg.top_k          # nothing speculates for layer 0
        for L in range(1, cfg.n_layers):
            want, dr = [], 0
            while len(want) < cfg.top_k:
                e = _spec_mix((t * cfg.n_layers + L) * 256 + dr) % cfg.n_experts
                dr += 1
                if e not in want:
                    want.append(e)
            assert pred[L].tolist() == want and len(set(want)) == cfg.top_k
            seen[want] += 1
        for L in range(cfg.n_layers):
            # within a step: layer L is used, then layer L + 1 is speculated
            if L >= 1:
                events[L].insert(len(events[L]), ("pred", pred[L].tolist()))
            events[L].append(("use", use[L].tolist()))
    assert seen.min() > 0
    hits = misses = pref = 0
    for L in range(cfg.n_layers):
        h, m, pf, order = _lru_sim(cfg.cache_slots, events[L], 3)
        hits += h; misses += m; pref += pf
        assert o.lru()[L].tolist() == order
    st = o.stats()
    assert (st["expert_hits"], st["expert_misses"], st["prefetched"]) == (hits, misses, pref)


def test_I23_previous_layer_speculation_is_the_next_router_on_h():
    """Policy 4 (L242: speculation from the previous layer's residual; L244: one layer ahead; Q25): the
    predicted experts of layer L+1 are route(W_r^{L+1}, rms(h_{L+1}; g2_{L+1})) with h_{L+1} the slow residual entering
    that layer, recomputed here in numpy from trace_h; counters equal the brute-force LRU simulation."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    P, steps = 5, 8
    o = Oracle(cfg, W)
    o.set_policy(4)
    o.prefill(S.gen_prompt(cfg, P))
    events = {L: [] for L in range(cfg.n_layers)}
    agree = 0
    for s in range(steps):
        o.decode_step()
        H, pred, use = o.trace_h(), o.pred_idx(), o.route_idx()
        for L in range(1, cfg.n_layers):
            g2 = S.as_f32(cfg, W["layers"][L]["g2"]).astype(np.float64)
            Wr = S.as_f32(cfg, W["layers"][L]["router"]).astype(np.float64)
            h = H[L].astype(np.float64)
            y = h / np.sqrt(np.mean(h * h) + cfg.rms_eps) * g2
            lg = Wr @ y
            want = list(np.argsort(-lg, kind="stable")[:cfg.top_k])
            assert pred[L].tolist() == [int(e) for e in want], (s, L)
            agree += len(set(want) & set(use[L].tolist()))
        for L in range(cfg.n_layers):
            if L >= 1:
                events[L].append(("pred", pred[L].tolist()))
            events[L].append(("use", use[L].tolist()))
    hits = misses = pref = 0
    for L in range(cfg.n_layers):
        h_, m_, pf, order = _lru_sim(cfg.cache_slots, events[L], 4)
        hits += h_; misses += m_; pref += pf
        assert o.lru()[L].tolist() == order
    st = o.stats()
    assert (st["expert_hits"], st["expert_misses"], st["prefetched"]) == (hits, misses, pref)
    # the previous-layer residual is an informative predictor (Fig. 9a): far above chance (top_k / n_e per slot)
    assert agree > 1.5 * steps * (cfg.n_layers - 1) * cfg.top_k * cfg.top_k / cfg.n_experts


def test_I18_moe_topk_mixture_bruteforce():
    """PAPER.md L131 / SURVEY §8(c).1 'MoE layer': h_{i+1} = h' + sum_{e in top-2} w_e Expert_e(rms(h'; g2)) with
    n_e = 8, top_k = 2 and RENORMALISED weights, against a numpy restatement (attention over the oracle's own
    cache, which I1/I6 pin).  Sensitivity: dropping the renormalisation or weighting both experts equally
    moves the result far outside the tolerance."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 7))
    for _ in range(3):
        o.decode_step()
        H = o.trace_h()
        t = o.kv_len - 1
        ri, rw = o.route_idx(), o.route_w()
        for i in range(cfg.n_layers):
            want, idx, w = np_moe_slow_layer(cfg, W["layers"][i], H[i], t, o.kcache(i), o.vcache(i))
            assert idx.tolist() == ri[i].tolist(), (i, idx, ri[i])
            assert idx[0] != idx[1]
            assert np.allclose(w, rw[i], atol=1e-6) and abs(w.sum() - 1.0) < 1e-12
            err = rel_l2(H[i + 1] - H[i], want - H[i])
            assert err < 5e-6, (i, err)
            # a plausible slip: un-renormalised softmax weights (sum < 1) or equal weights
            no_renorm, _, w_raw = np_moe_slow_layer(replace(cfg, renorm_topk=False), W["layers"][i], H[i], t,
                                                    o.kcache(i), o.vcache(i))
            assert w_raw.sum() < 0.9
            assert rel_l2(H[i + 1] - H[i], no_renorm - H[i]) > 1e-2


def test_I19_moe_accelerated_bottleneck_bruteforce():
    """PAPER.md L137 ('fixed set of accelerator adapters' while h takes the routed experts) in DESIGN Q7's
    reading: the accelerated stream of a MoE layer is attention-with-adapters followed by the rank-r_m SwiGLU
    bottleneck U_d(silu(U_g y^) * U_u y^), with NO expert involved.  Brute force in numpy from trace_p."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 6))
    for _ in range(2):
        o.decode_step()
        P = o.trace_p()
        t = o.kv_len - 1
        for i in range(cfg.n_layers):
            want = np_accel_layer_moe(cfg, W["layers"][i], P[i], t, o.kcache(i), o.vcache(i))
            assert rel_l2(P[i + 1] - P[i], want - P[i]) < 5e-6, i
            # sensitivity: gate and up swapped (silu on the wrong branch) is far off
            Lw = dict(W["layers"][i])
            Lw["Ug"], Lw["Uu"] = Lw["Uu"], Lw["Ug"]
            bad = np_accel_layer_moe(cfg, Lw, P[i], t, o.kcache(i), o.vcache(i))
            assert rel_l2(P[i + 1] - P[i], bad - P[i]) > 1e-3     # 200x the tolerance above
    # the accelerated stream of a MoE layer does not depend on the experts at all
    W2 = S.gen_weights(cfg)
    for L in W2["layers"]:
        for E in L["experts"]:
            E["ewd"][...] = 0
    o2 = Oracle(cfg, W2)
    o2.prefill(S.gen_prompt(cfg, 6))
    o2.decode_step()
    P2 = o2.trace_p()
    o3 = Oracle(cfg, W)
    o3.prefill(S.gen_prompt(cfg, 6))
    o3.decode_step()
    # layer 0 of the first decode step: p_0 = h_0 is the same embedding row and the layer-0 cache is identical
    assert np.array_equal(P2[1], o3.trace_p()[1])


def test_I20_expert_predictor_unscripted():
    """PAPER.md L387 / L137 in DESIGN Q16's reading: after accelerated layer i the experts of every target layer
    L' in targets(i) are predicted as top-2 of softmax(W_r^{L'} rms(p_{i+1}; g2_{L'})): the TARGET layer's router
    and the TARGET layer's g2, applied to the accelerated residual LEAVING layer i.  No router script, so the
    arithmetic itself decides.  The alternatives a slip would produce (source layer's g2, source layer's
    router, p entering the layer, the slow residual) must disagree somewhere, or the pin would be blind."""
    cfg = S.config_small_moe()
    assert cfg.aot_targets[0] == (2, 4) and cfg.aot_targets[1] == (4, 6)
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.set_policy(2)
    o.prefill(S.gen_prompt(cfg, 5))
    f = lambda a: S.as_f32(cfg, a).astype(np.float64)
    blind = {"g2_src": 0, "router_src": 0, "p_in": 0, "h": 0}
    checked = 0
    for _ in range(6):
        o.decode_step()
        P, H, pred = o.trace_p(), o.trace_h(), o.pred_idx()
        for i, (lo, hi) in enumerate(cfg.aot_targets):
            for Lt in range(lo, hi):
                Lw, Ls = W["layers"][Lt], W["layers"][i]
                idx, _ = np_route(cfg, f(Lw["router"]), np_rms(cfg, P[i + 1], f(Lw["g2"])))
                assert idx.tolist() == pred[Lt].tolist(), (i, Lt, idx, pred[Lt])
                checked += 1
                alts = {"g2_src": np_route(cfg, f(Lw["router"]), np_rms(cfg, P[i + 1], f(Ls["g2"])))[0],
                        "router_src": np_route(cfg, f(Ls["router"]), np_rms(cfg, P[i + 1], f(Lw["g2"])))[0],
                        "p_in": np_route(cfg, f(Lw["router"]), np_rms(cfg, P[i], f(Lw["g2"])))[0],
                        "h": np_route(cfg, f(Lw["router"]), np_rms(cfg, H[i + 1], f(Lw["g2"])))[0]}
                for k, v in alts.items():
                    blind[k] += int(v.tolist() != idx.tolist())
        untargeted = [L for L in range(cfg.n_layers) if not any(lo <= L < hi for lo, hi in cfg.aot_targets)]
        assert (pred[untargeted] == -1).all()
    assert checked == 6 * 4
    # the gains are 1 + 0.02 N(0,1): a wrong g2 rarely flips a top-2, so that alternative is only required
    # to be distinguishable through the router input norm; the others must flip at least once
    assert blind["router_src"] > 0 and blind["p_in"] > 0 and blind["h"] > 0, blind


def test_I20b_predictor_uses_target_layer_gain():
    """Same pin with gains that differ strongly between layers, so that taking g2 of the wrong layer flips
    the predicted experts."""
    cfg = S.config_small_moe()
    W = S.gen_weights(cfg)
    rng = np.random.default_rng(5)
    for L in W["layers"]:
        g = (1.0 + 0.9 * rng.standard_normal(cfg.d_model)).astype(np.float32)
        L["g2"][...] = (g.view(np.uint32) >> 16).astype(np.uint16)    # bf16 bits (truncation is fine: an input)
    o = Oracle(cfg, W)
    o.set_policy(2)
    o.prefill(S.gen_prompt(cfg, 5))
    f = lambda a: S.as_f32(cfg, a).astype(np.float64)
    flips = 0
    for _ in range(4):
        o.decode_step()
        P, pred = o.trace_p(), o.pred_idx()
        for i, (lo, hi) in enumerate(cfg.aot_targets):
            for Lt in range(lo, hi):
                Lw, Ls = W["layers"][Lt], W["layers"][i]
                idx, _ = np_route(cfg, f(Lw["router"]), np_rms(cfg, P[i + 1], f(Lw["g2"])))
                assert idx.tolist() == pred[Lt].tolist()
                flips += int(np_route(cfg, f(Lw["router"]), np_rms(cfg, P[i + 1], f(Ls["g2"])))[0].tolist() != idx.tolist())
    assert flips > 0


def test_I21_lm_head_adapter_on_exit_logits():
    """PAPER.md L162 ('low-rank layers for ... language modeling heads') in DESIGN Q9's reading: the exit / draft
    logits at a gate are W_lm z + B_lm (A_lm z) with z = rms(p_E; g_f), p_E the accelerated residual BEFORE the
    gate reset; the final head on h never takes the adapter.  numpy from trace_p / trace_h."""
    cfg = tiny(lm_head_adapter=True)
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    o.prefill(S.gen_prompt(cfg, 9))
    f = lambda a: S.as_f32(cfg, a).astype(np.float64)
    for _ in range(3):
        o.decode_step()
        P, H = o.trace_p(), o.trace_h()
        E = cfg.gates[0]
        z = np_rms(cfg, P[E], f(W["gf"]))
        base = f(W["lm_head"]) @ z
        want = base + f(W["lm_B"]) @ (f(W["lm_A"]) @ z)
        got = o.exit_logits(0)
        assert rel_l2(got, want) < 2e-6
        assert rel_l2(got, base) > 1e-3            # the adapter is live: leaving it out is visible
        zh = np_rms(cfg, H[cfg.n_layers], f(W["gf"]))
        assert rel_l2(o.logits(), f(W["lm_head"]) @ zh) < 2e-6     # final head: no adapter
    # a draft taken through spec_step uses the same head
    o.spec_step(2)
    # with the flag off the same weights give the base logits
    o2 = Oracle(replace(cfg, lm_head_adapter=False), {k: v for k, v in W.items() if k not in ("lm_A", "lm_B")})
    o2.prefill(S.gen_prompt(cfg, 9))
    o2.decode_step()
    z2 = np_rms(cfg, o2.trace_p()[cfg.gates[0]], f(W["gf"]))
    assert rel_l2(o2.exit_logits(0), f(W["lm_head"]) @ z2) < 2e-6
