"""GPU-vs-oracle comparison helpers (tests only)."""
import numpy as np

import m2r2_synth as S
from tests.refs import rel_l2

MARGIN = 1e-3   # BASELINE.json: tokens must match except where the oracle's top-2 margin < 1e-3


def tolerances(cfg):
    """BASELINE.json north_star: fp32 tiny rel-L2 <= 1e-4; bf16 hidden rel-L2 <= 1e-2 and
    logits max-abs <= 5e-2."""
    if cfg.dtype == S.FP32:
        return dict(hidden=1e-4, logits_rel=1e-4, logits_abs=None)
    return dict(hidden=1e-2, logits_rel=None, logits_abs=5e-2)


def check_logits(cfg, got, want, what=""):
    tol = tolerances(cfg)
    if tol["logits_rel"] is not None:
        assert rel_l2(got, want) <= tol["logits_rel"], (what, rel_l2(got, want))
    if tol["logits_abs"] is not None:
        assert float(np.max(np.abs(got - want))) <= tol["logits_abs"], (what, float(np.max(np.abs(got - want))))


def check_hidden(cfg, got, want, what=""):
    """Per-layer hidden state: rel-L2 within the tolerance north_star states, AND a max-abs bound of the same
    relative size against the largest element, so that a single wrong row among thousands (which a norm over
    the whole vector would hide) fails: a wrong row is off by about the typical magnitude, i.e. ~0.25 of the
    largest element, against a bound of 1e-2 (bf16) / 1e-4 (fp32) of it."""
    tol = tolerances(cfg)["hidden"]
    e = rel_l2(got, want)
    assert e <= tol, (what, e)
    worst = float(np.max(np.abs(np.asarray(got, np.float64) - np.asarray(want, np.float64))))
    scale = float(np.max(np.abs(want)))
    assert worst <= 4.0 * tol * max(scale, 1e-30), (what, "max-abs", worst, scale)
    return e


def compare_decode_step(cfg, eng, orc, dbg, b=0, check_exit=True):
    """After both sides ran the SAME (teacher-forced) decode step: compare every h_i, p_i,
    the logits, the greedy token and the exit tokens."""
    H, P = orc.trace_h(), orc.trace_p()
    worst = 0.0
    for i in range(cfg.n_layers + 1):
        eh = check_hidden(cfg, eng.debug_read(dbg.DBG_H, i, b), H[i], ("h", i))
        ep = check_hidden(cfg, eng.debug_read(dbg.DBG_P, i, b), P[i], ("p", i))
        worst = max(worst, eh, ep)
    check_logits(cfg, eng.debug_read(dbg.DBG_LOGITS, 0, b), orc.logits(), "final logits")
    return worst
