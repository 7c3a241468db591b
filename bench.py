#!/usr/bin/env python
"""bench.py -- throughput of the per-GPU MoE-layer hot path (route -> permute -> grouped
SwiGLU FFN -> combine) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C1]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is ONE pass of the whole hot path over one batch of synthetic input (BASELINE.json
configs[1], the Mixtral-8x7B-shaped layer, unless --config says otherwise).  `value` is
whole-job tokens/s with inputs resident in HBM; `e2e` is the same metric through the C-ABI
call that takes HOST buffers (H2D of logits+X and D2H of out+counts inside the timed region).
N > 1: independent replicas, one per GPU, no data-path collective.
--impl reference: the CPU oracle (oracle/), as it stands, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "moe_layer_tokens_per_s"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                    "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"]))}, "measured"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback"


def load_ncu_traffic(config_name: str):
    """DRAM bytes (read + write) per vibe_grouped_ffn call (both launches) from the committed
    `ncu --set full` capture, or None.  profiles/ffn_traffic.csv: config,dram_bytes,source."""
    p = os.path.join(ROOT, "profiles", "ffn_traffic.csv")
    if os.path.exists(p):
        try:
            for ln in open(p):
                cols = [c.strip() for c in ln.split(",")]
                if len(cols) >= 2 and cols[0] == config_name:
                    return float(cols[1])
        except Exception:
            return None
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reason_bits, self.power = [], 0, []
        self._stop_evt = threading.Event()
        self.max_mhz = None
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.reason_bits |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                self.power.append(self.nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        out = {"sm_mhz": int(statistics.median(self.samples)) if self.samples else None,
               "sm_max_mhz": self.max_mhz,
               "reasons": [n for b, n in sorted(self.REASONS.items()) if self.reason_bits & b],
               "samples": len(self.samples)}
        if self.power:
            out["power_w_max"] = round(max(self.power), 1)
        return out


def oracle_sample_step(O, I, cfg, L, S):
    """The whole hot path in the oracle on the first S tokens of a batch."""
    lg, X = L["logits"][:S], L["X"][:S]
    ids, w, counts = O.route_topk(lg, select_bias=L["select_bias"], **I.route_kwargs(cfg))
    em = L["expert_map"] if cfg.E_loc < cfg.E else None
    off, r2a, a2r, Xp, R = O.permute(X, ids, em, cfg.E_loc, 1)
    Y, _ = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    out = O.combine(Y, a2r, w, S, cfg.k, round_out=True)
    return out, int((np.diff(off) > 0).sum())


def run_reference(args, group):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only)."""
    if not group.is_main:
        return
    from oracle import vibe_oracle as O
    from paper_2606_00735_b200 import inputs as I
    cfg = I.CONFIGS[args.config]
    L = I.make_layer(cfg, args.seed)
    cores = len(os.sched_getaffinity(0))
    # bounded sample: per step the oracle converts every touched expert's bf16 weights to f64
    # (~3*d*f elements each); choose the largest S whose estimated cost fits the step budget
    t0 = time.perf_counter()
    O.bf16_bits_to_f64(L["W1"][0])
    per_expert = 3.3 * (time.perf_counter() - t0) + 6.0 * cfg.d * cfg.f * 8 / 20e9
    # The whole run must end within a few minutes.  A step can not cost less than one token
    # (k experts' weights converted to f64), so when K+W such steps do not fit, fewer steps are
    # run and the line reports the count actually timed.
    total_budget = 200.0
    min_step = min(cfg.E_loc, cfg.k) * per_expert
    steps = max(1, min(args.steps, int(total_budget * 0.8 / min_step)))
    warmup = max(0, min(args.warmup, int(total_budget * 0.2 / min_step)))
    budget = total_budget / (steps + warmup)
    S = 1
    for cand in (2, 4, 8, 16, 32, 64, 128, 256):
        touched = min(cfg.E_loc, cand * cfg.k)
        if cand <= cfg.T and touched * per_expert <= budget:
            S = cand
    for _ in range(warmup):
        oracle_sample_step(O, I, cfg, L, S)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_sample_step(O, I, cfg, L, S)
    dt = time.perf_counter() - t0
    requested = (args.steps, args.warmup)
    args.steps, args.warmup = steps, warmup
    value = S * args.steps / dt
    sample = f"first {S} of {cfg.T} tokens per step through oracle route+permute+grouped_ffn+combine (fp64 numpy)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "T": cfg.T, "d": cfg.d, "f": cfg.f, "E": cfg.E, "k": cfg.k,
                   "E_loc": cfg.E_loc, "sample_tokens_per_step": S,
                   "steps_requested": requested[0], "warmup_requested": requested[1]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=40)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C1", choices=["C0", "C1", "C2", "C3"])
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--sets", type=int, default=4, help="rotating input buffer sets")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_2606_00735_b200 import dist as D
    if args.impl == "reference":
        world = int(os.environ.get("WORLD_SIZE", "1"))
        if world > 1 and int(os.environ.get("RANK", "0")) != 0:
            return                      # other ranks exit 0 without work
        run_reference(args, D.Group(0, 1, 0, None))
        return

    import torch
    from paper_2606_00735_b200 import binding as B
    from paper_2606_00735_b200 import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU fallback (use --impl reference "
                         "for the oracle)")
    group = D.init_from_env()
    torch.cuda.set_device(group.local_rank)
    dev = torch.device("cuda", group.local_rank)
    B.load()
    cfg = I.CONFIGS[args.config]
    peaks, peak_kind = load_peaks()

    # ---------------------------------------------------------------- inputs (seeded, numpy)
    def pin_bf16(shape):
        return torch.empty(shape, dtype=torch.bfloat16).pin_memory()

    Wh = [pin_bf16((cfg.E_loc, cfg.d, cfg.f)), pin_bf16((cfg.E_loc, cfg.d, cfg.f)), pin_bf16((cfg.E_loc, cfg.f, cfg.d))]
    I.make_weights(cfg.E_loc, cfg.d, cfg.f, args.seed,
                   out=[w.view(torch.int16).numpy().view(np.uint16) for w in Wh])
    W1, W3, W2 = (w.to(dev, non_blocking=True) for w in Wh)
    emap_np = I.make_expert_map(cfg, "contiguous", args.seed)
    emap = torch.from_numpy(emap_np).to(dev) if cfg.E_loc < cfg.E else None
    bias_np = I.make_select_bias(cfg.E, args.seed) if cfg.has_select_bias else None
    bias = torch.from_numpy(bias_np).to(dev) if bias_np is not None else None
    rc = B.RouteConfig(select_bias=bias, **I.route_kwargs(cfg))
    sets_h, sets_d = [], []
    for i in range(args.sets):
        lg = torch.from_numpy(I.make_logits(cfg.T, cfg.E, cfg.zipf_s, args.seed + i, cfg.alpha)).pin_memory()
        Xb = torch.from_numpy(I.make_X(cfg.T, cfg.d, args.seed + i).view(np.int16)).view(torch.bfloat16).pin_memory()
        sets_h.append((lg, Xb))
        sets_d.append((lg.to(dev), Xb.to(dev)))
    T, k, E, E_loc, d, f = cfg.T, cfg.k, cfg.E, cfg.E_loc, cfg.d, cfg.f
    A = T * k
    Rcap = max(1, B.rows_cap(T, k, E_loc, 1))
    ids = torch.empty((T, k), dtype=torch.int32, device=dev)
    gw = torch.empty((T, k), dtype=torch.float32, device=dev)
    counts = torch.empty((E,), dtype=torch.int32, device=dev)
    Xp = torch.empty((Rcap, d), dtype=torch.bfloat16, device=dev)
    H = torch.empty((Rcap, f), dtype=torch.bfloat16, device=dev)
    Y = torch.empty((Rcap, d), dtype=torch.bfloat16, device=dev)
    off = torch.empty((E_loc + 1,), dtype=torch.int32, device=dev)
    r2a = torch.empty((Rcap,), dtype=torch.int32, device=dev)
    a2r = torch.empty((A,), dtype=torch.int32, device=dev)
    out = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
    pws = torch.empty((max(16, B.workspace_bytes(B.WS_PERMUTE, T, k, E, E_loc, d, f)),), dtype=torch.uint8, device=dev)
    fws = torch.empty((max(16, B.workspace_bytes(B.WS_FFN, T, k, E, E_loc, d, f)),), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step(i, ev=None):
        lg, Xd = sets_d[i % args.sets]
        if ev:
            ev[0].record(stream)
        B.route_topk(lg, rc, out=(ids, gw, counts), stream=stream)
        if ev:
            ev[1].record(stream)
        B.permute(Xd, ids, counts, emap, E, E_loc, 1, out=(Xp, off, r2a, a2r), ws=pws, stream=stream)
        if ev:
            ev[2].record(stream)
        B.grouped_ffn(Xp, off, W1, W3, W2, H=H, Y=Y, stream=stream, ws=fws)
        if ev:
            ev[3].record(stream)
        B.combine(Y, a2r, gw, T, k, out=out, stream=stream)
        if ev:
            ev[4].record(stream)

    # ---------------------------------------------------------------- device-resident timing
    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(group.local_rank)
    group.barrier()
    torch.cuda.synchronize()
    sampler.start()
    n0 = B.launch_count()
    t_start.record(stream)
    for i in range(args.steps):
        step(i, evs[i])
    t_end.record(stream)
    torch.cuda.synchronize()
    launches = B.launch_count() - n0
    clocks = sampler.stop()
    group.barrier()
    my_ms = t_start.elapsed_time(t_end)
    value, max_ms = D.aggregate_throughput(group, float(T) * args.steps, my_ms)
    stage_ms = [sum(e[j].elapsed_time(e[j + 1]) for e in evs) / args.steps for j in range(4)]

    # real rows / resident tokens of the routed batches (for algorithmic bytes and flops): the buffer sets differ
    # when only a shard of the experts is resident, so average over the sets in the proportion they were used
    R_set, tok_set, rows_per_expert = [], [], []
    for i in range(args.sets):
        step(i)
        torch.cuda.synchronize()
        R_set.append(int(off[-1].item()))
        rows_per_expert += torch.diff(off).tolist()
        tok_set.append(int((a2r.view(T, k) >= 0).any(dim=1).sum().item()))
    uses = [len(range(i, args.steps, args.sets)) for i in range(args.sets)]
    R_real = sum(r * u for r, u in zip(R_set, uses)) / max(1, sum(uses))
    res_tok = sum(r * u for r, u in zip(tok_set, uses)) / max(1, sum(uses))

    # ---------------------------------------------------------------- end to end from host buffers
    # Through vibe_moe_layer_forward_host_async / vibe_host_wait, the call a serving loop makes: every step copies its
    # logits + X from pinned host memory and its result + counts back, inside the timed region.  Steps are issued
    # back to back on two arenas / two result buffers, so step i+1's copy-in and step i-1's copy-out overlap step
    # i's kernels; a step's result is waited for before its arena is reused (two steps later).
    nbuf = 2
    arenas = [torch.empty((B.workspace_bytes(B.WS_LAYER_HOST, T, k, E, E_loc, d, f),), dtype=torch.uint8, device=dev)
              for _ in range(nbuf)]
    outs_h = [torch.empty((T, d), dtype=torch.bfloat16).pin_memory() for _ in range(nbuf)]
    cnts_h = [torch.empty((E,), dtype=torch.int32).pin_memory() for _ in range(nbuf)]

    def run_e2e(n):
        tickets = [None] * nbuf
        for i in range(n):
            b = i % nbuf
            if tickets[b] is not None:
                B.host_wait(tickets[b])
            tickets[b] = B.moe_layer_forward_host_async(rc, *sets_h[i % args.sets], emap, W1, W3, W2, outs_h[b], cnts_h[b],
                                                        arenas[b], stream=stream)
        for tk in tickets:
            if tk is not None:
                B.host_wait(tk)

    run_e2e(3)
    # the asynchronous entry returns the bits of the device-resident entry on the same batch (the synchronous host
    # entry cuts the batch into chunks, and a chunk's last round of FFN tiles may take the split-K path: same
    # values, another summation order)
    ref_d, refc_d = B.moe_layer_forward(rc, *sets_d[2 % args.sets], emap, W1, W3, W2, arena=arenas[0], stream=stream)
    torch.cuda.synchronize()
    e2e_same_bits = bool(torch.equal(ref_d.cpu().view(torch.int16), outs_h[2 % nbuf].view(torch.int16)) and
                         torch.equal(refc_d.cpu(), cnts_h[2 % nbuf]))
    del ref_d, refc_d
    group.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    run_e2e(args.steps)              # returns after the last result has arrived on the host
    e1.record(stream)
    torch.cuda.synchronize()
    group.barrier()
    e2e_value, _ = D.aggregate_throughput(group, float(T) * args.steps, e0.elapsed_time(e1))
    h2d = T * E * 4 + T * d * 2
    d2h = T * d * 2 + E * 4
    del arenas

    # ---------------------------------------------------------------- the same layer with the FP8 (e4m3) FFN (S8(f) f2)
    # extra information, not the headline: BASELINE.json's configs are bf16.  Weights are quantised once, outside
    # the timed region (they are static in serving); the activations are quantised inside it.
    fp8 = None
    if d % 128 == 0 and f % 128 == 0:
        def time_layer(fn, n):
            for i in range(max(3, args.warmup // 4)):
                fn(i)
            torch.cuda.synchronize()
            a8, b8 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a8.record(stream)
            for i in range(n):
                fn(i)
            b8.record(stream)
            torch.cuda.synchronize()
            return a8.elapsed_time(b8) / n

        n8 = max(20, args.steps // 2)
        cnt8 = torch.empty((E,), dtype=torch.int32, device=dev)
        # (i) block-scaled e4m3 (readings Q5-Q8: UE8M0 scale per row and 32 K elements, applied by the tensor core)
        W1m, sf13 = B.mxfp8_pack_weights(W1, B.MX_ROLE_GATE)
        W3m, sf13 = B.mxfp8_pack_weights(W3, B.MX_ROLE_UP, sf=sf13)
        W2m, sf2 = B.mxfp8_pack_weights(W2, B.MX_ROLE_DOWN)
        arena_mx = torch.empty((B.workspace_bytes(B.WS_LAYER_MXFP8, T, k, E, E_loc, d, f),), dtype=torch.uint8, device=dev)
        ms_mx = time_layer(lambda i: B.moe_layer_forward_mxfp8(rc, *sets_d[i % args.sets], emap, W1m, W3m, sf13, W2m, sf2,
                                                               out=out, counts=cnt8, arena=arena_mx, stream=stream), n8)
        del W1m, W3m, W2m, arena_mx
        # (ii) per-expert / per-row scales (Q1-Q4).  The static scale of the intermediate is CALIBRATED on this
        # workload: 2 x the largest |H| per expert of the bf16 path on batch 0, / 448; the fraction of H codes that
        # sit on the saturation value in a step is reported
        step(0)
        torch.cuda.synchronize()
        offs = off.tolist()
        hs8 = torch.tensor([2.0 * float(H[offs[e]:offs[e + 1]].abs().max()) / 448.0 if offs[e + 1] > offs[e] else 1.0
                            for e in range(E_loc)], dtype=torch.float32, device=dev).clamp_min(1e-6)
        W1q, s1q = B.fp8_pack_weights(W1)
        W3q, s3q = B.fp8_pack_weights(W3)
        W2q, s2q = B.fp8_pack_weights(W2)
        la = B.workspace_bytes(B.WS_LAYER_FP8, T, k, E, E_loc, d, f)
        arena8 = torch.empty((la,), dtype=torch.uint8, device=dev)
        ms8 = time_layer(lambda i: B.moe_layer_forward_fp8(rc, *sets_d[i % args.sets], emap, W1q, s1q, W3q, s3q, W2q, s2q,
                                                           hs8, out=out, counts=cnt8, arena=arena8, stream=stream), n8)
        fp8 = {"mxfp8_layer_tokens_per_s": round(T / ms_mx * 1e3), "mxfp8_ms_per_step": round(ms_mx, 4),
               "layer_tokens_per_s": round(T / ms8 * 1e3), "ms_per_step": round(ms8, 4), "steps": n8,
               "note": "mxfp8 = vibe_moe_layer_forward_mxfp8 (block-scaled e4m3, UE8M0 scale per 32 K elements); the other pair = "
                       "vibe_moe_layer_forward_fp8 (per-expert / per-row scales, h_scale calibrated: 2 x max|H| of batch 0 / 448); "
                       "one rank; parity of both at this size: tests/test_gpu_full_size.py"}
        del W1q, W3q, W2q, arena8

    # ---------------------------------------------------------------- roofline of the dominant kernel
    # The peak follows from the evidence of THIS run: a timed region that stayed near the maximum SM clock
    # with no power cap is a burst-clock measurement (denominator: the burst cuBLAS figure); a run the
    # power cap throttled is held against the sustained figure.  Both fractions are printed.
    ffn_s = stage_ms[2] * 1e-3
    flops = 6.0 * R_real * d * f
    achieved_tf = flops / ffn_s / 1e12
    sustained, burst = peaks["bf16_tflops_sustained"], peaks["bf16_tflops"]
    mhz, mhz_max = clocks.get("sm_mhz"), clocks.get("sm_max_mhz")
    capped = "sw_power_cap" in clocks.get("reasons", []) and mhz is not None and mhz_max and mhz < 0.9 * mhz_max
    peak, why = (sustained, f"sustained: sw_power_cap seen, median SM clock {mhz} of {mhz_max} MHz") if capped else \
                (burst, f"burst: median SM clock {mhz} of {mhz_max} MHz, not throttled by the power cap")
    hbm = peaks["hbm_gbs"]
    # S8(d): per expert max(flops / tensor peak, bytes / HBM peak), summed -- the bound that applies to skewed routing
    bound_s = 0.0
    for n in rows_per_expert:
        if n > 0:
            bound_s += max(6.0 * n * d * f / (peak * 1e12), (6.0 * d * f + 2.0 * n * d + 4.0 * n * f + 2.0 * n * d) / (hbm * 1e9))
    bound_s /= max(1, args.sets)
    roofline = {"kernel": "ffn_gemm_kernel (2 launches per step: gate_up+SwiGLU, down)", "bound": "tensor",
                "achieved": round(achieved_tf, 2), "peak": peak, "unit": "TFLOP/s",
                "frac": round(achieved_tf / peak, 4),
                "traffic": load_ncu_traffic(cfg.name),
                "traffic_source": "committed ncu --set full capture (profiles/ffn_traffic.csv), not this run",
                "peak_kind": f"{peak_kind} cuBLAS bf16, {why}",
                "frac_of_burst": round(achieved_tf / burst, 4), "frac_of_sustained": round(achieved_tf / sustained, 4),
                "per_expert_bound_ms": round(bound_s * 1e3, 4),
                "frac_of_per_expert_bound": round(bound_s / ffn_s, 4),
                "flops_per_step": flops, "ms_per_step": round(stage_ms[2], 4)}
    bytes_route = 4.0 * T * E + 8.0 * T * k + 4.0 * E
    bytes_perm = 2.0 * res_tok * d + 2.0 * R_real * d + 12.0 * A
    bytes_comb = 2.0 * R_real * d + 2.0 * T * d + 8.0 * A
    # in-step event pairs sit between Python-issued launches: for the microsecond-scale stages they time the
    # host's launch pace, so they carry no roofline fraction (the alone_* fields below do)
    stages = {}
    for name, ms in (("route", stage_ms[0]), ("permute", stage_ms[1]), ("combine", stage_ms[3])):
        stages[name] = {"in_step_ms_host_paced": round(ms, 4)}
    stages["grouped_ffn"] = {"ms": round(stage_ms[2], 4), "TFLOP/s": round(achieved_tf, 2)}

    # ---------------------------------------------------------------- bandwidth kernels alone, from CUDA graphs
    # The per-stage events above sit between Python-issued launches, so for the microsecond-scale
    # route / permute / combine stages they mostly time the host.  Here each stage is captured
    # (one call per rotating buffer set) into a CUDA graph and replayed: device time only.
    def graph_us(fn, reps=20):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for i in range(args.sets):
                fn(i)
        g.replay()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            g.replay()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e3 / (reps * args.sets)

    iso = {
        "route": graph_us(lambda i: B.route_topk(sets_d[i % args.sets][0], rc, out=(ids, gw, counts))),
        "permute": graph_us(lambda i: B.permute(sets_d[i % args.sets][1], ids, counts, emap, E, E_loc, 1,
                                                out=(Xp, off, r2a, a2r), ws=pws)),
        "combine": graph_us(lambda i: B.combine(Y, a2r, gw, T, k, out=out)),
    }
    for name, by in (("route", bytes_route), ("permute", bytes_perm), ("combine", bytes_comb)):
        gbs = by / (iso[name] * 1e-6) / 1e9
        stages[name].update({"alone_us": round(iso[name], 2), "alone_GB/s": round(gbs, 1),
                             "alone_frac_hbm": round(gbs / hbm, 4)})

    # ---------------------------------------------------------------- CPU baseline (oracle, rank 0, N = 1)
    cpu_baseline = None
    if group.is_main and group.world == 1 and not args.no_cpu_baseline:
        from oracle import vibe_oracle as O
        S = min(T, 512)
        L = {"logits": sets_h[0][0].numpy(), "X": sets_h[0][1].view(torch.int16).numpy().view(np.uint16),
             "select_bias": bias_np, "expert_map": emap_np,
             "W1": Wh[0].view(torch.int16).numpy().view(np.uint16),
             "W3": Wh[1].view(torch.int16).numpy().view(np.uint16),
             "W2": Wh[2].view(torch.int16).numpy().view(np.uint16)}
        t0 = time.perf_counter()
        ref_out, touched = oracle_sample_step(O, I, cfg, L, S)
        dt = time.perf_counter() - t0
        cpu_baseline = {"value": S / dt, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
                        "sample": f"first {S} of {T} tokens of batch 0 through the fp64 numpy oracle "
                                  f"(route+permute+grouped_ffn+combine, {touched} experts touched), {dt:.1f} s"}

    if group.is_main:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": group.world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": cfg.name, "T": T, "d": d, "f": f, "E": E, "k": k, "E_loc": E_loc,
                       "routing": f"zipf_s={cfg.zipf_s} alpha={cfg.alpha}", "real_rows": round(R_real, 1),
                       "real_rows_per_set": R_set,
                       "parallelism": "replicas" if group.world > 1 else "single-gpu",
                       "l2": f"inputs rotate over {args.sets} buffer sets; "
                             f"{(3 * E_loc * d * f * 2) / 1e9:.2f} GB of weights stream through the 126 MB L2 every step"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "entry": "vibe_moe_layer_forward_host_async + vibe_host_wait, 2 arenas in flight, pinned host buffers",
                    "same_bits_as_device_entry": e2e_same_bits},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "stages": stages,
            "ffn_tflops": round(achieved_tf, 2),
            "fp8": fp8,
        }
        print(json.dumps(line), flush=True)
    group.close()


if __name__ == "__main__":
    main()
