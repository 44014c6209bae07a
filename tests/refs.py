"""Independent references used to PIN the oracle (never used by the product).

`torch_decoder` is a textbook pre-norm decoder (RMSNorm, rotate-half RoPE, causal SDPA,
SwiGLU) assembled from torch CPU library ops over the FULL sequence — the special case the
M2R2 slow stream must reduce to (Eq. 1 L47-50 with the norms of footnote 1 L60;
BASELINE.json invariant 1).  `np_accel_layer` is a brute-force dense restatement of the
accelerated layer (Eq. 2, attention L76) that builds the (t+1)-row key/value
matrices [K[0..t-1]; k^_t] explicitly.
"""
import numpy as np
import torch
import torch.nn.functional as F

import m2r2_synth as S


def _t(cfg, a):
    return torch.from_numpy(S.as_f32(cfg, a).astype(np.float64))


def _round_bf16(x):
    return x.to(torch.float32).to(torch.bfloat16).to(torch.float64)


def _rotate_half(x):
    h = x.shape[-1] // 2
    return torch.cat((-x[..., h:], x[..., :h]), dim=-1)


def torch_decoder(cfg, W, tokens):
    """-> (hidden [N+1, T, d], logits [T, V]) in float64, slow stream only."""
    T = len(tokens)
    nh, dh, d = cfg.n_heads, cfg.head_dim, cfg.d_model
    x = _t(cfg, W["embed"])[torch.as_tensor(np.asarray(tokens), dtype=torch.long)]
    pos = torch.arange(T, dtype=torch.float64)
    inv_freq = cfg.rope_theta ** (-torch.arange(0, dh, 2, dtype=torch.float64) / dh)
    ang = torch.outer(pos, inv_freq)
    cos = torch.cat((ang.cos(), ang.cos()), dim=-1)[None]
    sin = torch.cat((ang.sin(), ang.sin()), dim=-1)[None]
    hidden = [x]
    for L in W["layers"]:
        xn = x * torch.rsqrt(x.pow(2).mean(-1, keepdim=True) + cfg.rms_eps) * _t(cfg, L["g1"])
        q = (xn @ _t(cfg, L["wq"]).T).view(T, nh, dh).transpose(0, 1)
        k = (xn @ _t(cfg, L["wk"]).T).view(T, nh, dh).transpose(0, 1)
        v = (xn @ _t(cfg, L["wv"]).T).view(T, nh, dh).transpose(0, 1)
        # torch ops above run in fp64; the oracle rounds each projection to fp32 first
        q = q * cos + _rotate_half(q) * sin
        k = k * cos + _rotate_half(k) * sin
        if cfg.dtype == S.BF16:
            k, v = _round_bf16(k), _round_bf16(v)
        o = F.scaled_dot_product_attention(q[None], k[None], v[None], is_causal=True)[0]
        x = x + o.transpose(0, 1).reshape(T, d) @ _t(cfg, L["wo"]).T
        xn = x * torch.rsqrt(x.pow(2).mean(-1, keepdim=True) + cfg.rms_eps) * _t(cfg, L["g2"])
        x = x + (F.silu(xn @ _t(cfg, L["wgate"]).T) * (xn @ _t(cfg, L["wup"]).T)) @ _t(cfg, L["wdown"]).T
        hidden.append(x)
    xn = x * torch.rsqrt(x.pow(2).mean(-1, keepdim=True) + cfg.rms_eps) * _t(cfg, W["gf"])
    logits = xn @ _t(cfg, W["lm_head"]).T
    return torch.stack(hidden).numpy(), logits.numpy()


def np_rms(cfg, x, g):
    x = x.astype(np.float64)
    return x / np.sqrt((x * x).mean() + cfg.rms_eps) * g


def np_rope(cfg, v, t):
    dh = cfg.head_dim
    half = dh // 2
    v = v.astype(np.float64).reshape(-1, dh).copy()
    j = np.arange(half)
    ang = t * cfg.rope_theta ** (-2.0 * j / dh)
    a, b = v[:, :half].copy(), v[:, half:].copy()
    v[:, :half] = a * np.cos(ang) - b * np.sin(ang)
    v[:, half:] = b * np.cos(ang) + a * np.sin(ang)
    return v.reshape(-1)


def np_accel_layer(cfg, Lw, p, t, Kc, Vc, h=None, topk=0):
    """Brute-force accelerated layer for a dense model.  Kc/Vc: slow cache [>=t, d].
    topk > 0: per head the accelerated query attends only the `topk` cached positions with the
    largest SLOW attention scores (slow query of the same token = rope(W_q rms(h; g1)) with `h` the slow residual
    entering the layer; ties: lower position) plus its own key."""
    f = lambda k: S.as_f32(cfg, Lw[k]).astype(np.float64)
    dh = cfg.head_dim
    Sh = list(cfg.accel_heads)
    rows = np.concatenate([np.arange(a * dh, (a + 1) * dh) for a in Sh])
    x = np_rms(cfg, p, f("g1"))
    q = f("wq")[rows] @ x + f("Bq") @ (f("Aq") @ x)
    k = f("wk")[rows] @ x + f("Bk") @ (f("Ak") @ x)
    v = f("wv")[rows] @ x + f("Bv") @ (f("Av") @ x)
    q, k = np_rope(cfg, q, t), np_rope(cfg, k, t)
    o = np.zeros(len(rows))
    for s, a in enumerate(Sh):
        sl = slice(s * dh, (s + 1) * dh)
        Kmat = np.vstack([Kc[:t, a * dh:(a + 1) * dh].astype(np.float64), k[sl][None]])   # (t+1, dh)
        Vmat = np.vstack([Vc[:t, a * dh:(a + 1) * dh].astype(np.float64), v[sl][None]])
        sc = Kmat @ q[sl] / np.sqrt(dh)
        if topk and t > topk:
            qs = np_rope(cfg, (f("wq") @ np_rms(cfg, h, f("g1"))).astype(np.float32), t)[a * dh:(a + 1) * dh].astype(np.float64)
            ss = Kc[:t, a * dh:(a + 1) * dh].astype(np.float64) @ qs / np.sqrt(dh)
            chosen = sorted(range(t), key=lambda u: (-ss[u], u))[:topk]
            mask = np.full(t + 1, -np.inf)
            mask[chosen] = 0.0
            mask[t] = 0.0
            sc = sc + mask
        pr = np.exp(sc - sc.max())
        pr /= pr.sum()
        o[sl] = pr @ Vmat
    p1 = p.astype(np.float64) + f("wo")[:, rows] @ o + f("Bo") @ (f("Ao") @ o)
    y = np_rms(cfg, p1, f("g2"))
    g = f("wgate") @ y + f("Bg") @ (f("Ag") @ y)
    u = f("wup") @ y + f("Bu") @ (f("Au") @ y)
    a_ = g / (1 + np.exp(-g)) * u
    return p1 + f("wdown") @ a_ + f("Bd") @ (f("Ad") @ a_)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-30))


# ---------------------------------------------------------------------------------------------
# Brute-force restatements of the MoE / predictor / LM-head-adapter branches (pins I18-I21).
# Written from PAPER.md and DESIGN.md's readings in numpy float64; they share nothing with oracle/.
# ---------------------------------------------------------------------------------------------
def np_route(cfg, Wr, y, renorm=True):
    """Router (DESIGN Q19): softmax over ALL experts, the top_k largest (lower index
    first on ties), weights renormalised over the selected ones.  -> (idx[top_k], w[top_k])"""
    logits = Wr.astype(np.float64) @ y.astype(np.float64)
    pr = np.exp(logits - logits.max())
    pr /= pr.sum()
    order = sorted(range(len(pr)), key=lambda e: (-pr[e], e))[:cfg.top_k]
    w = pr[order]
    if renorm:
        w = w / w.sum()
    return np.asarray(order, dtype=np.int32), w


def np_swiglu(Wg, Wu, Wd, y):
    g, u = Wg @ y, Wu @ y
    return Wd @ (g / (1.0 + np.exp(-g)) * u)


def np_slow_attention(cfg, Lw, h, t, Kc, Vc):
    """h' = h + W_o concat_a softmax(q_a K_a[0..t]^T / sqrt(dh)) V_a[0..t]  (Eq. 1) for the token at
    position t, given the slow cache INCLUDING position t (the cache itself is pinned by I1 / I6)."""
    f = lambda k: S.as_f32(cfg, Lw[k]).astype(np.float64)
    dh, nh = cfg.head_dim, cfg.n_heads
    x = np_rms(cfg, h, f("g1"))
    q = np_rope(cfg, (f("wq") @ x).astype(np.float32), t)
    o = np.zeros(cfg.d_model)
    for a in range(nh):
        sl = slice(a * dh, (a + 1) * dh)
        sc = Kc[:t + 1, sl].astype(np.float64) @ q[sl] / np.sqrt(dh)
        pr = np.exp(sc - sc.max())
        pr /= pr.sum()
        o[sl] = pr @ Vc[:t + 1, sl].astype(np.float64)
    return h.astype(np.float64) + f("wo") @ o


def np_moe_slow_layer(cfg, Lw, h, t, Kc, Vc):
    """Slow MoE layer: attention as above, then m = sum_{e in top-k} w_e Expert_e(rms(h'; g2))
    (SURVEY §8(c).1 'MoE layer').  -> (h_{i+1}, idx, w)"""
    f = lambda a: S.as_f32(cfg, a).astype(np.float64)
    h1 = np_slow_attention(cfg, Lw, h, t, Kc, Vc)
    y = np_rms(cfg, h1, f(Lw["g2"]))
    idx, w = np_route(cfg, f(Lw["router"]), y, cfg.renorm_topk)
    m = np.zeros(cfg.d_model)
    for e, we in zip(idx, w):
        E = Lw["experts"][int(e)]
        m += we * np_swiglu(f(E["ewg"]), f(E["ewu"]), f(E["ewd"]), y)
    return h1 + m, idx, w


def np_accel_layer_moe(cfg, Lw, p, t, Kc, Vc):
    """Accelerated layer of a MoE model: attention with adapters as in the dense case, then the FIXED
    adapter-only bottleneck  m^ = U_d (silu(U_g y^) * (U_u y^))  (DESIGN Q7)."""
    f = lambda k: S.as_f32(cfg, Lw[k]).astype(np.float64)
    dh = cfg.head_dim
    Sh = list(cfg.accel_heads)
    rows = np.concatenate([np.arange(a * dh, (a + 1) * dh) for a in Sh])
    x = np_rms(cfg, p, f("g1"))
    q = f("wq")[rows] @ x + f("Bq") @ (f("Aq") @ x)
    k = f("wk")[rows] @ x + f("Bk") @ (f("Ak") @ x)
    v = f("wv")[rows] @ x + f("Bv") @ (f("Av") @ x)
    q, k = np_rope(cfg, q, t), np_rope(cfg, k, t)
    o = np.zeros(len(rows))
    for s, a in enumerate(Sh):
        sl = slice(s * dh, (s + 1) * dh)
        Kmat = np.vstack([Kc[:t, a * dh:(a + 1) * dh].astype(np.float64), k[sl][None]])
        Vmat = np.vstack([Vc[:t, a * dh:(a + 1) * dh].astype(np.float64), v[sl][None]])
        sc = Kmat @ q[sl] / np.sqrt(dh)
        pr = np.exp(sc - sc.max())
        pr /= pr.sum()
        o[sl] = pr @ Vmat
    p1 = p.astype(np.float64) + f("wo")[:, rows] @ o + f("Bo") @ (f("Ao") @ o)
    y = np_rms(cfg, p1, f("g2"))
    return p1 + np_swiglu(f("Ug"), f("Uu"), f("Ud"), y)
