#!/usr/bin/env python
"""bench.py — M2R2 decode throughput on B200 (contract: see DESIGN.md §Measurement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W
    python bench.py --workload c3|c4|c5|olmoe|gemma [--gamma G] [--alpha A] [--tokens T]     # secondary workloads

Workload of the bench line (BASELINE.json configs[1], "C2"): 3.8B-class bf16 decoder (32 layers, d 3072, 32x96 heads,
FFN 8192, vocab 32064), batch 1, 512-token random prompt, then K dual-stream M2R2 decode steps (slow
and accelerated residual streams both carried through all 32 layers).  A "step" = one
m2r2_decode_step = one generated token.  Synthetic seeded weights N(0, 0.02) and uniform-random
prompt (m2r2_synth).  N > 1 = N independent replicas (no collective).

Prints ONE JSON line (rank 0).  `value` is device-timed (CUDA events on the library's compute
stream, inputs resident in HBM, tokens stay on the device); `e2e` is the same metric through the C
ABI with host buffers (the forced input token goes host->device, the produced token device->host,
every step, inside the timed region).  `roofline` is for the dominant kernel class measured live by
the library's event profile; `selfspec` is the metric's other half, the same model under self-speculative
decoding (BASELINE.json configs[2], "C3": gamma 4, acceptance 0.9 and 0.5, 256 tokens, device-timed over the whole
generation), `selfspec_batch8` the batched case (configs[3], "C4": 8 sequences x 4096-token KV, gamma 4, acceptance 0.9, 48
spec_steps); `cpu_baseline` is the oracle timed on this box's host cores.
`--impl reference` times the oracle (CPU) on the same config and metric.

Secondary workloads (one JSON line each): c3 = self-spec sweep (gamma x alpha), c4 = batch 8 x 4096-token KV self-spec,
c5 = MoE expert-loading policies with copy/compute overlap accounting, olmoe = the paper's five strategies on an
OLMoE-shaped model, gemma = self-spec on a Gemma-7B-class shape (f-4).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "decode tokens/s at batch 1 (M2R2 self-spec); achieved HBM GB/s vs 8 TB/s"   # BASELINE.json wording
PROMPT = 512
HBM_NOMINAL_GBS = 8000.0      # BASELINE.json: "achieved HBM GB/s vs 8 TB/s"
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of m2r2_fused_decode_kernel (one decode step at
# kv_len ~ 521) from the committed capture profiles/r2_v33_fused_kernel.md (ncu --set full): 7.690 GB + 21.8 MB
FUSED_TRAFFIC_BYTES = 7.690290e9 + 21.755648e6


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------
# byte model (DESIGN.md §Byte model): algorithmic bytes one decode step must move
# ---------------------------------------------------------------------------------------------
def step_bytes(cfg, T, exit_heads):
    """T = positions already cached (kv_len before the step)."""
    e, d, F, r = cfg.elt_bytes, cfg.d_model, cfg.d_ff, cfg.adapter_rank
    da = cfg.n_accel_heads * cfg.head_dim
    w_layer = (4 * d * d + 3 * d * F) * e
    ad_layer = (3 * (r * d + da * r) + r * da + d * r + 2 * (r * d + F * r) + r * F + d * r) * e
    n_acc = cfg.accel_end_layer if cfg.accel_enabled else 0
    by = {"qkv": cfg.n_layers * 3 * d * d * e + n_acc * 3 * (r * d + da * r) * e,
          "o_proj": cfg.n_layers * d * d * e + n_acc * (r * da + d * r) * e,
          "gate_up": cfg.n_layers * 2 * d * F * e + n_acc * 2 * (r * d + F * r) * e,
          "down": cfg.n_layers * d * F * e + n_acc * (r * F + d * r) * e,
          "attention": cfg.n_layers * 2 * d * (T + 1) * e,
          "rope_append": cfg.n_layers * 2 * d * e,
          "heads": (1 + (len(cfg.gates) if exit_heads else 0)) * cfg.vocab * d * e,
          "other": d * e}
    total = sum(by.values())
    assert total == cfg.n_layers * w_layer + n_acc * ad_layer + by["attention"] + by["rope_append"] + by["heads"] + by["other"]
    return total, by


# ---------------------------------------------------------------------------------------------
# clocks (B200_PROFILING.md): nvidia-smi sampled DURING the timed region
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1]))
                mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference): oracle/ as it stands, host cores
# ---------------------------------------------------------------------------------------------
def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def time_oracle(cfg, W, n_steps, warmup, prefill_tokens=8, budget_s=None):
    """Oracle decode steps on the C2 model after a short prefill.  A 3.8B decode step streams the
    same 7.6 GB of weights whatever the context length (KV is 2.6% of the bytes at T=512), so a
    short context is a fair bounded sample of the workload.  -> (tokens/s, steps timed, description)"""
    import m2r2_synth as S
    from oracle import Oracle
    orc = Oracle(cfg, W)
    orc.prefill(S.gen_prompt(cfg, prefill_tokens))
    t_first = None
    for _ in range(max(1, warmup)):
        t0 = time.perf_counter()
        orc.decode_step()
        t_first = time.perf_counter() - t0
    if budget_s is not None and t_first * n_steps > budget_s:
        n_steps = max(2, int(budget_s / t_first))
    t0 = time.perf_counter()
    for _ in range(n_steps):
        orc.decode_step()
    dt = time.perf_counter() - t0
    orc.close()
    desc = ("%d oracle decode steps of the C2 model (all 32 layers, both streams) at context %d..%d after a "
            "%d-token prefill and %d warm-up steps" % (n_steps, prefill_tokens + max(1, warmup),
                                                      prefill_tokens + max(1, warmup) + n_steps,
                                                      prefill_tokens, max(1, warmup)))
    return n_steps / dt, n_steps, dt, desc


def bench_config():
    import m2r2_synth as S
    return S.config_c2()


def config_json(cfg, extra=None):
    c = {"workload": "C2 (BASELINE.json configs[1]): 3.8B-class bf16 dense decoder, batch 1, prompt %d, "
                     "plain M2R2 dual-stream decode steps (slow + accelerated stream in all %d layers, "
                     "accel heads %d of %d, adapter rank %d, gates %s re-initialise p from h)"
                     % (PROMPT, cfg.n_layers, cfg.n_accel_heads, cfg.n_heads, cfg.adapter_rank, list(cfg.gates)),
         "n_layers": cfg.n_layers, "d_model": cfg.d_model, "n_heads": cfg.n_heads, "head_dim": cfg.head_dim,
         "d_ff": cfg.d_ff, "vocab": cfg.vocab, "batch": 1, "prompt_len": PROMPT,
         "l2_policy": "inputs larger than L2: every step streams >= 7.6 GB of weights + KV (L2 is 126 MB)",
         "parallelism": "replicas"}
    if extra:
        c.update(extra)
    return c


def run_reference(args, rk):
    """--impl reference: the oracle on host cores, same config / metric / unit (tier framing ④)."""
    from paper_2502_02040_b200 import replicas
    if rk.rank != 0:
        return 0
    import m2r2_synth as S
    cfg = bench_config()
    W = S.gen_weights(cfg)
    tps, n, dt, desc = time_oracle(cfg, W, args.steps, args.warmup, budget_s=150.0)
    line = {"impl": "reference", "metric": METRIC, "value": tps, "unit": "tokens/s", "n_gpus": args.gpus,
            "steps": n, "steps_requested": args.steps, "warmup": max(1, args.warmup),
            "ms_per_step": 1e3 * dt / n, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 arithmetic with f64 accumulation (bf16 weights + KV)", "data": "synthetic",
            "config": config_json(cfg),
            "cpu_baseline": {"value": tps, "unit": "tokens/s", "cores": host_cores(), "kind": "oracle", "sample": desc},
            "e2e": {"value": tps, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args, rk):
    import torch
    import m2r2_synth as S
    import paper_2502_02040_b200 as M
    from paper_2502_02040_b200 import replicas

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    dev = "cuda:%d" % rk.local_rank
    torch.cuda.set_device(dev)
    cfg = bench_config()
    K, Wm = args.steps, max(3, args.warmup)
    if PROMPT + 2 * (Wm + K) + 8 > cfg.max_seq:
        from dataclasses import replace
        cfg = replace(cfg, max_seq=PROMPT + 2 * (Wm + K) + 8)
    exit_heads = bool(args.exit_heads)
    W = S.gen_weights(cfg)
    eng = M.Engine(cfg, W, exit_heads=exit_heads, device=dev)
    if args.no_fused:
        eng.set_fused(False)
    prompt = S.gen_prompt(cfg, PROMPT, seed=replicas.replica_seed(1000 + 2, rk))
    stream = eng.compute_stream
    peak, peak_src = measured_peaks()

    def timed_device(n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n):
            eng.decode_step(want_tokens=False)      # token stays on the device
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1)

    # ---- device-timed region: K steps, inputs resident in HBM
    eng.prefill(prompt)
    for _ in range(Wm):
        eng.decode_step(want_tokens=False)
    eng.sync()
    launches0 = eng.get_stats()["kernel_launches"]
    kv0 = eng.get_stats()["kv_len"][0]
    replicas.barrier(rk)
    torch.cuda.synchronize()
    clocks = ClockSampler(rk.local_rank) if rk.rank == 0 else None
    ms = timed_device(K)
    torch.cuda.synchronize()
    replicas.barrier(rk)
    clk = clocks.stop() if clocks else None
    launches = eng.get_stats()["kernel_launches"] - launches0
    ms_max, units = replicas.aggregate(rk, ms, K)
    value = units / (ms_max * 1e-3)

    # ---- algorithmic bytes of the timed steps (T grows kv0 .. kv0+K-1)
    tot_bytes = sum(step_bytes(cfg, kv0 + s, exit_heads)[0] for s in range(K))
    step_gbs = tot_bytes / (ms * 1e-3) / 1e9
    lib_bytes = eng.get_stats()["algorithmic_bytes_last"]
    model_last = step_bytes(cfg, kv0 + K - 1, exit_heads)[0]
    assert abs(lib_bytes - model_last) <= 1e-6 * model_last, (lib_bytes, model_last)

    # ---- per-class profile pass (same steps, events between kernel groups) -> dominant kernel roofline
    eng.prefill(prompt)
    for _ in range(Wm):
        eng.decode_step(want_tokens=False)
    eng.set_profile(True)
    n_prof = min(K, 32)
    for _ in range(n_prof):
        eng.decode_step(want_tokens=False)
    prof = eng.get_profile()
    eng.set_profile(False)
    _, by_cls = step_bytes(cfg, kv0 + n_prof // 2, exit_heads)
    per_class = {}
    for c, t_ms in prof["ms"].items():
        b = tot_bytes / K if c == "fused_step" else by_cls.get(c, 0)
        per_class[c] = {"ms_per_step": t_ms, "launch_groups_per_step": prof["segments"][c],
                        "algorithmic_bytes_per_step": b, "GB/s": b / (t_ms * 1e-3) / 1e9 if t_ms > 0 else None}
    dom = max(prof["ms"], key=lambda c: prof["ms"][c])
    dom_groups = prof["segments"][dom]
    dom_bytes = per_class[dom]["algorithmic_bytes_per_step"] / dom_groups
    dom_ms = prof["ms"][dom] / dom_groups
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
    kernel_names = {"gate_up": "gemv_kernel<bf16, 2 rows, SWIGLU> (+ norm_lora_kernel)", "qkv": "gemv_kernel<bf16, 2 rows> (+ norm_lora_kernel)",
                    "down": "gemv_kernel<bf16, 2 rows>", "o_proj": "gemv_kernel<bf16, 2 rows>", "heads": "gemv_kernel<bf16> LM head",
                    "attention": "attn_kernel + merge_kernel", "fused_step": "m2r2_fused_decode_kernel (persistent, whole step)"}
    roofline = {"bound": "hbm", "kernel": kernel_names.get(dom, dom), "class": dom,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "peak_source": peak_src, "bytes_per_launch": dom_bytes, "ms_per_launch": dom_ms,
                "traffic": args.traffic if dom == "fused_step" else None,
                "traffic_source": "profiles/r2_v33_fused_kernel.md (ncu --set full, one launch)" if dom == "fused_step" else None,
                "step": {"achieved": step_gbs, "frac": step_gbs / peak,
                                                  "frac_of_nominal_8TBs": step_gbs / HBM_NOMINAL_GBS,
                                                  "algorithmic_bytes_per_step": tot_bytes / K},
                "per_class": per_class}

    # ---- e2e: same metric through the C ABI with HOST buffers, one H2D + one D2H per step
    first = eng.prefill(prompt)
    tok = np.array([int(first[0])], dtype=np.int32)
    for _ in range(Wm):
        tok = eng.decode_step(force_tokens=tok)
    replicas.barrier(rk)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(K):
        tok = eng.decode_step(force_tokens=tok)      # host token in (H2D), host token out (D2H + sync)
    e1.record(stream)
    e1.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = max(e0.elapsed_time(e1), wall_ms)
    e2e_max, e2e_units = replicas.aggregate(rk, e2e_ms, K)
    e2e = {"value": e2e_units / (e2e_max * 1e-3), "unit": "tokens/s", "h2d_bytes_per_step": 4, "d2h_bytes_per_step": 4,
           "ms_per_step": e2e_max / K}

    line = {"metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": rk.world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 arithmetic (bf16 weights + KV cache)", "data": "synthetic",
            "config": config_json(cfg),
            "run": {"exit_heads_at_gates": exit_heads, "kv_len_start": kv0,
                    "implementation": "per-operation kernels" if args.no_fused else "default",
                    "value_is": "plain M2R2 dual-stream decode steps of C2 (the workload the roofline target is stated on); "
                                "the self-speculative tokens/s of the same model are in `selfspec`"},
            "clocks": clk, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline}

    # ---- cpu_baseline: oracle on this box's host cores (rank 0, N = 1 only)
    eng.close()
    del eng
    torch.cuda.empty_cache()
    if rk.rank == 0 and rk.world == 1 and not args.no_selfspec:
        line["selfspec"] = selfspec_record(peak)
        torch.cuda.empty_cache()
        line["selfspec_batch8"] = selfspec_batch8_record(peak)
        torch.cuda.empty_cache()
    if rk.rank == 0 and rk.world == 1 and not args.no_cpu_baseline:
        tps, n, dt, desc = time_oracle(cfg, W, 12, 1, budget_s=25.0)
        line["cpu_baseline"] = {"value": tps, "unit": "tokens/s", "cores": host_cores(), "kind": "oracle", "sample": desc}
    if rk.rank == 0:
        print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# self-speculative decoding of the same 3.8B model (BASELINE.json configs[2], "C3"): the metric's "M2R2 self-spec"
# ---------------------------------------------------------------------------------------------
def selfspec_record(peak, gamma=4, alphas=(0.9, 0.5), n_tokens=256):
    """C3: drafts from the accelerated stream at layer 8 (gamma draft passes of layers 0..7 + draft head), one
    gamma+1-token verify pass of the full model with greedy acceptance and KV rollback, acceptance forced to alpha
    by the seeded logit script.  Device-timed (CUDA events on the library's compute stream) over the
    whole generation of n_tokens tokens after a 512-token prompt; spec_step returns the accepted tokens to the host
    every step, so this is also the end-to-end number."""
    import torch
    import m2r2_synth as S
    import paper_2502_02040_b200 as M
    cfg = S.config_c3()
    eng = M.Engine(cfg, S.gen_weights(cfg), device="cuda:0")
    prompt = S.gen_prompt(cfg, PROMPT)
    stream = eng.compute_stream
    rec = {"workload": "C3 (BASELINE.json configs[2]): the C2 model under self-speculative decoding, drafts from the "
                       "accelerated stream at layer 8 (E = 8, LM-head adapter rank 8), draft length gamma = %d, "
                       "prompt %d, %d generated tokens, acceptance forced by seeded logit biasing" % (gamma, PROMPT, n_tokens),
           "gamma": gamma, "runs": []}
    for alpha in alphas:
        f, g = S.gen_logit_script(cfg, n_tokens + 160, alpha)
        eng.set_logit_script(f, g, PROMPT)
        eng.prefill(prompt)
        for _ in range(3):
            eng.spec_step(gamma)
        eng.prefill(prompt)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        emitted, steps, by = 1, 0, 0
        l0 = eng.get_stats()["kernel_launches"]
        e0.record(stream)
        while emitted < n_tokens:
            _, n = eng.spec_step(gamma)
            emitted += int(n[0])
            steps += 1
            by += eng.get_stats()["algorithmic_bytes_last"]
        e1.record(stream)
        e1.synchronize()
        ms = e0.elapsed_time(e1)
        gbs = by / (ms * 1e-3) / 1e9
        rec["runs"].append({"alpha": alpha, "tokens": emitted - 1, "spec_steps": steps, "tokens_per_s": (emitted - 1) / (ms * 1e-3),
                            "ms_per_spec_step": ms / steps, "tokens_per_spec_step": (emitted - 1) / steps,
                            "algorithmic_bytes_per_spec_step": by / steps, "GB/s": gbs, "frac_of_measured_peak": gbs / peak,
                            "frac_of_nominal_8TBs": gbs / HBM_NOMINAL_GBS,
                            "gpu_launches_per_spec_step": (eng.get_stats()["kernel_launches"] - l0) / steps})
    eng.set_logit_script(None, None, PROMPT)
    eng.prefill(prompt)
    for _ in range(3):
        eng.decode_step(want_tokens=False)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(128):
        eng.decode_step(want_tokens=False)
    e1.record(stream)
    e1.synchronize()
    rec["plain_decode_control_tokens_per_s"] = 128 / (e0.elapsed_time(e1) * 1e-3)
    eng.close()
    return rec


def selfspec_batch8_record(peak, gamma=4, alpha=0.9, n_steps=48):
    """C4 (BASELINE.json configs[3]): the same model, 8 sequences x 4096-token KV, spec_step(4) with per-sequence seeded logit
    scripts at acceptance alpha; the batched passes run on the tensor-core GEMM / attention kernels.  Device-timed over
    n_steps spec_steps (every step returns its accepted tokens to the host)."""
    import torch
    import m2r2_synth as S
    import paper_2502_02040_b200 as M
    cfg = S.config_c4()
    B, P = 8, 4096
    eng = M.Engine(cfg, S.gen_weights(cfg), device="cuda:0")
    stream = eng.compute_stream
    prompts = np.stack([S.gen_prompt(cfg, P, seq=b) for b in range(B)])
    scripts = [S.gen_logit_script(cfg, 8 * (n_steps + 8), alpha, seq=b) for b in range(B)]
    eng.set_logit_script(np.stack([x[0] for x in scripts]), np.stack([x[1] for x in scripts]), P)
    eng.prefill(prompts)
    for _ in range(3):
        eng.spec_step(gamma)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    emitted, by = 0, 0
    l0 = eng.get_stats()["kernel_launches"]
    e0.record(stream)
    for _ in range(n_steps):
        _, n = eng.spec_step(gamma)
        emitted += int(n.sum())
        by += eng.get_stats()["algorithmic_bytes_last"]
    e1.record(stream)
    e1.synchronize()
    ms = e0.elapsed_time(e1)
    gbs = by / (ms * 1e-3) / 1e9
    rec = {"workload": "C4 (BASELINE.json configs[3]): the C3 model, batch 8, 4096-token KV per sequence, draft length gamma = %d, "
                       "acceptance %.1f forced by per-sequence seeded logit biasing, %d spec_steps" % (gamma, alpha, n_steps),
           "gamma": gamma, "alpha": alpha, "batch": B, "kv_len_start": P, "spec_steps": n_steps,
           "aggregate_tokens_per_s": emitted / (ms * 1e-3), "ms_per_spec_step": ms / n_steps,
           "tokens_per_spec_step": emitted / n_steps, "algorithmic_bytes_per_spec_step": by / n_steps, "GB/s": gbs,
           "frac_of_measured_peak": gbs / peak, "frac_of_nominal_8TBs": gbs / HBM_NOMINAL_GBS,
           "gpu_launches_per_spec_step": (eng.get_stats()["kernel_launches"] - l0) / n_steps}
    eng.close()
    return rec


# ---------------------------------------------------------------------------------------------
# secondary workloads (BASELINE.json configs[2..4]); not the driver's bench line: `--workload c3|c4|c5`
# ---------------------------------------------------------------------------------------------
def run_secondary(args):
    """C3 self-spec (gamma x alpha), C4 batch-8 long-KV self-spec, C5 MoE expert loading policies.
    Wall-clock around synchronised library calls (each call returns host results, so it is the e2e number)."""
    import torch
    import m2r2_synth as S
    import paper_2502_02040_b200 as M
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    out = {"workload": args.workload, "data": "synthetic", "n_gpus": 1, "runs": []}
    if args.workload in ("c3", "gemma"):
        # gemma: SURVEY 8(f) f-4, the paper's self-spec regime (Gemma-7B-class shape, E = 4, gamma = 3)
        cfg = S.config_c3() if args.workload == "c3" else S.config_gemma7b_class()
        out["model"] = cfg.name
        eng = M.Engine(cfg, S.gen_weights(cfg), device="cuda:0")
        prompt = S.gen_prompt(cfg, PROMPT)
        for alpha in ((args.alpha,) if args.alpha else (0.9, 0.5)):
            for gamma in ((args.gamma,) if args.gamma else ((2, 4, 6) if args.workload == "c3" else (3,))):
                f, g = S.gen_logit_script(cfg, 400, alpha)
                eng.set_logit_script(f, g, PROMPT)
                eng.prefill(prompt)
                for _ in range(3):
                    eng.spec_step(gamma)
                eng.prefill(prompt)
                torch.cuda.synchronize()
                torch.cuda.profiler.start()     # `ncu --profile-from-start off` captures the timed region only
                t0, emitted, steps, by = time.perf_counter(), 1, 0, 0
                while emitted < args.tokens:
                    _, n = eng.spec_step(gamma)
                    emitted += int(n[0])
                    steps += 1
                    by += eng.get_stats()["algorithmic_bytes_last"]
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
                torch.cuda.profiler.stop()
                out["runs"].append({"alpha": alpha, "gamma": gamma, "tokens": emitted - 1, "spec_steps": steps,
                                    "ms_per_spec_step": 1e3 * dt / steps, "tokens_per_s": (emitted - 1) / dt,
                                    "tokens_per_spec_step": (emitted - 1) / steps, "algorithmic_GB_per_s": by / dt / 1e9})
        eng.set_logit_script(None, None, PROMPT)
        eng.prefill(prompt)
        for _ in range(3):
            eng.decode_step()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(128):
            eng.decode_step()
        torch.cuda.synchronize()
        out["plain_decode_control_tokens_per_s"] = 128 / (time.perf_counter() - t0)
        eng.close()
    elif args.workload == "c4":
        cfg = S.config_c4()
        B, P, gamma = 8, 4096, 4
        eng = M.Engine(cfg, S.gen_weights(cfg), device="cuda:0")
        prompts = np.stack([S.gen_prompt(cfg, P, seq=b) for b in range(B)])
        for alpha in ((args.alpha,) if args.alpha else (0.9, 0.5)):
            scripts = [S.gen_logit_script(cfg, 1000, alpha, seq=b) for b in range(B)]
            eng.set_logit_script(np.stack([x[0] for x in scripts]), np.stack([x[1] for x in scripts]), P)
            eng.prefill(prompts)
            for _ in range(2):
                eng.spec_step(gamma)
            torch.cuda.synchronize()
            nsteps = 128 if args.tokens == 256 else args.tokens     # --tokens N: N spec steps (short profiled runs)
            torch.cuda.profiler.start()     # `ncu --profile-from-start off` captures the timed region only
            t0, emitted, by = time.perf_counter(), 0, 0
            for _ in range(nsteps):
                _, n = eng.spec_step(gamma)
                emitted += int(n.sum())
                by += eng.get_stats()["algorithmic_bytes_last"]
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            torch.cuda.profiler.stop()
            out["runs"].append({"alpha": alpha, "gamma": gamma, "batch": B, "kv_len_start": P, "spec_steps": nsteps,
                                "ms_per_spec_step": 1e3 * dt / nsteps, "aggregate_tokens_per_s": emitted / dt,
                                "algorithmic_GB_per_s": by / dt / 1e9, "kv_len_end": list(eng.get_stats()["kv_len"][:B])})
        eng.close()
    else:
        from dataclasses import replace
        base = S.config_c5()
        P, STEPS = 256, 256 if args.tokens == 256 else args.tokens
        eng0 = M.Engine(base, device="cuda:0")
        # one weight set for every scenario: generated for the widest accelerated range (layers 0..7 carry adapters; a
        # config whose accelerated stream ends earlier ignores the rest); expert store in pinned host memory (kept by eng0)
        W = S.gen_weights(replace(base, gates=(8,), accel_end_layer=8), expert_alloc=eng0.pinned_expert_alloc())
        prompt = S.gen_prompt(base, P)
        # the link: pinned host -> device copy of one expert blob, best of 5 (what a load costs at best)
        ebytes = 3 * base.d_model * base.d_ff_expert * 2
        src = torch.empty(ebytes, dtype=torch.uint8).pin_memory()
        dst = torch.empty(ebytes, dtype=torch.uint8, device="cuda:0")
        best = 1e9
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); dst.copy_(src, non_blocking=True); e1.record(); e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        link_gbs = ebytes / (best * 1e-3) / 1e9
        out["h2d_link_GB_per_s"] = link_gbs
        out["expert_bytes"] = ebytes
        del src, dst

        def run(eng, pol, rho, pi):
            act, pred = S.gen_router_script(eng.cfg, P + STEPS + 44, rho, pi)
            eng.set_policy(pol)
            eng.set_router_script(act, pred, 0)
            eng.prefill(prompt)
            for _ in range(4):
                eng.decode_step()
            s0 = eng.get_stats()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(STEPS):
                eng.decode_step()
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            s1 = eng.get_stats()
            d = {k: s1[k] - s0[k] for k in ("expert_hits", "expert_misses", "expert_prefetched", "expert_on_demand", "h2d_bytes")}
            return dt, d

        scenarios = [("C5 as BASELINE.json states it: 2 slots per layer, p_4 predicts layers 4..15", base, 0.25, 0.9),
                     ("perfect predictor (pi = 1.0)", base, 0.25, 1.0),
                     ("the paper's 2x schedule, layer i predicts {2i+2, 2i+3} (PAPER.md L137, L244, L387)",
                      replace(base, gates=(8,), accel_end_layer=8, aot_targets=S.aot_targets_for_rate(base.n_layers, 2, 8)), 0.25, 0.9),
                     ("4 slots per layer (half of the experts resident, the paper's ratio L242)", replace(base, cache_slots=4), 0.25, 0.9)]
        for name, cfg, rho, pi in scenarios:
            eng = eng0 if cfg is base else M.Engine(cfg, device="cuda:0")
            if eng is not eng0 or not getattr(eng0, "_loaded", False):
                eng.load_weights(W)
                eng._loaded = True
            # compute-only reference: every step routes the same pair (rho = 1): all hits after the first step
            dt_c, _ = run(eng, M.POLICY_LRU, 1.0, 1.0)
            comp_ms = 1e3 * dt_c / STEPS
            for pol, pname in ((M.POLICY_FIXED, "on-demand"), (M.POLICY_LRU, "LRU"), (M.POLICY_LRU_AOT, "LRU+AoT")):
                dt, d = run(eng, pol, rho, pi)
                ms = 1e3 * dt / STEPS
                copy_ms = d["h2d_bytes"] / STEPS / (link_gbs * 1e9) * 1e3      # time the step's loads need on the link at its best
                hidden = max(0.0, comp_ms + copy_ms - ms)                      # what ran concurrently
                out["runs"].append({"scenario": name, "policy": pname, "router_script": {"rho": rho, "pi": pi}, "steps": STEPS,
                                    "cache_slots": cfg.cache_slots, "ms_per_step": ms, "tokens_per_s": STEPS / dt,
                                    "hit_rate": d["expert_hits"] / max(1, d["expert_hits"] + d["expert_misses"]),
                                    "prefetched": d["expert_prefetched"], "on_demand": d["expert_on_demand"],
                                    "h2d_GB": d["h2d_bytes"] / 1e9, "h2d_GB_per_s": d["h2d_bytes"] / 1e9 / dt,
                                    "compute_only_ms_per_step": comp_ms, "link_ms_per_step_at_peak": copy_ms,
                                    "overlap_ms_per_step": hidden,
                                    "overlap_fraction_of_compute": hidden / comp_ms if comp_ms > 0 else None})
            if eng is not eng0:
                eng.close()
        eng0.close()
    print(json.dumps(out), flush=True)
    return 0


def run_olmoe(args):
    """the paper's five expert-loading strategies on an OLMoE-shaped model with half of
    the experts resident, natural (un-scripted) routing of the random-init routers.  Reports per-step latency (Fig. 9b's
    metric), hit rate at use (Fig. 9a's), bytes loaded and the link rate."""
    import torch
    import m2r2_synth as S
    import paper_2502_02040_b200 as M
    cfg = S.config_olmoe_shaped()
    P, STEPS = 64, 128 if args.tokens == 256 else args.tokens
    eng = M.Engine(cfg, device="cuda:0")
    W = S.gen_weights(cfg, expert_alloc=eng.pinned_expert_alloc())
    eng.load_weights(W)
    prompt = S.gen_prompt(cfg, P)
    out = {"workload": "olmoe-shaped (f-2)", "data": "synthetic", "n_gpus": 1, "config": {"n_layers": cfg.n_layers, "d_model": cfg.d_model,
           "n_experts": cfg.n_experts, "top_k": cfg.top_k, "d_ff_expert": cfg.d_ff_expert, "cache_slots_per_layer": cfg.cache_slots,
           "expert_bytes": 3 * cfg.d_model * cfg.d_ff_expert * 2, "aot_schedule": "layer i -> {2i+2, 2i+3}, i < 8"}, "runs": []}
    names = {M.POLICY_FIXED: "fixed + on-demand", M.POLICY_LRU: "LRU", M.POLICY_LRU_RANDOM: "LRU + random speculation",
             M.POLICY_LRU_PREV: "LRU + previous-layer residual", M.POLICY_LRU_AOT: "LRU + accelerated residual (M2R2 AoT)"}
    # random-init routers on random-init hidden states pick almost the same experts every step (LRU hit rate 0.995), so
    # two of the eight routed experts per layer and step follow the seeded router script (reused from the previous step
    # with probability rho = 0.25, predicted correctly with probability pi = 0.9); the other six stay natural
    act, pred = S.gen_router_script(cfg, P + STEPS + 44, 0.25, 0.9)
    out["router_script"] = {"rho": 0.25, "pi": 0.9, "scripted_experts_per_layer": 2}
    for pol in (M.POLICY_FIXED, M.POLICY_LRU, M.POLICY_LRU_RANDOM, M.POLICY_LRU_PREV, M.POLICY_LRU_AOT):
        eng.set_policy(pol)
        eng.set_router_script(act, pred, 0)
        eng.prefill(prompt)
        for _ in range(4):
            eng.decode_step()
        s0 = eng.get_stats()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(STEPS):
            eng.decode_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        s1 = eng.get_stats()
        d = {k: s1[k] - s0[k] for k in ("expert_hits", "expert_misses", "expert_prefetched", "expert_on_demand", "h2d_bytes")}
        out["runs"].append({"policy": names[pol], "steps": STEPS, "ms_per_step": 1e3 * dt / STEPS, "tokens_per_s": STEPS / dt,
                            "hit_rate_at_use": d["expert_hits"] / max(1, d["expert_hits"] + d["expert_misses"]),
                            "prefetched": d["expert_prefetched"], "on_demand": d["expert_on_demand"],
                            "h2d_GB": d["h2d_bytes"] / 1e9, "h2d_GB_per_s": d["h2d_bytes"] / 1e9 / dt})
    eng.close()
    print(json.dumps(out), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=256)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--exit-heads", type=int, default=0, help="evaluate the exit argmax at every gate (SURVEY Q15 second row)")
    ap.add_argument("--no-fused", action="store_true", help="force the per-operation kernels")
    ap.add_argument("--workload", default="c2", choices=["c2", "c3", "c4", "c5", "olmoe", "gemma"],
                    help="c2 = the bench line (default); c3/c4/c5 = secondary workloads of BASELINE.json configs[2..4]; "
                         "olmoe = the five expert-loading strategies on an OLMoE-shaped model (SURVEY 8(f) f-2); gemma = self-spec on a "
                         "Gemma-7B-class shape, E = 4, gamma = 3 (f-4)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gamma", type=int, default=0, help="--workload c3: one draft length instead of 2, 4, 6")
    ap.add_argument("--alpha", type=float, default=0.0, help="--workload c3: one acceptance rate instead of 0.9, 0.5")
    ap.add_argument("--tokens", type=int, default=256, help="--workload c3: tokens to generate per run")
    ap.add_argument("--no-selfspec", action="store_true", help="skip the C3 self-speculative sub-record of the bench line")
    ap.add_argument("--traffic", type=float, default=FUSED_TRAFFIC_BYTES,
                    help="dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/)")
    args = ap.parse_args()
    if args.workload == "olmoe":
        sys.exit(run_olmoe(args))
    if args.workload != "c2":
        sys.exit(run_secondary(args))
    from paper_2502_02040_b200 import replicas
    rk = replicas.init_from_env(backend="gloo" if args.impl == "reference" else None)
    if args.gpus != rk.world and rk.world > 1:
        raise SystemExit("--gpus %d but WORLD_SIZE %d" % (args.gpus, rk.world))
    try:
        rc = run_reference(args, rk) if args.impl == "reference" else run_ours(args, rk)
    finally:
        replicas.shutdown(rk)
    sys.exit(rc)


if __name__ == "__main__":
    main()
