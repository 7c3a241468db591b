"""Per-kernel measurements on one B200 beyond the single bench.py line.

    python -m paper_2606_00735_b200.report [--sections stages,ffn,mixed,fp8,fused,layer,profile,placement,variability,rack,recalibration]
                                           [--out gpurun_out/report.json] [--quick]

Sections (all through the C-ABI binding; seeded synthetic inputs):
  stages     route / permute / combine timed one kernel family at a time on rotating buffer
             sets whose footprint exceeds the 126 MB L2 (cold reads), for BASELINE.json
             configs[1..3] and a 64K-token stress shape: achieved GB/s = algorithmic bytes
              / CUDA-event time, and the fraction of the measured HBM peak.
  ffn        grouped FFN on BALANCED routing (every expert n rows), n = 128..4096, for the
             C1/C2/C3 shapes: TFLOP/s and fraction of the measured bf16 peaks -- the
             ">= 512 tokens per expert" target of BASELINE.json is read off this table.
  fp8        vibe_grouped_ffn_fp8 (e4m3 operands) next to the bf16 kernel, balanced routing.
  fused      vibe_grouped_ffn + vibe_combine versus the fused gate-weighted scatter path
             (vibe_grouped_ffn_scatter + vibe_combine_scattered) on the routed C1 / C2 batches.
  layer      the whole layer through vibe_moe_layer_forward, eager launches versus one CUDA graph.
  profile    vibe_profile_expert_latency over the M3 sweep (1..4096 tokens per expert), modes 0
             and 1, for the C2 and C3 shapes: the per-GPU performance model f(n) of the paper
             (PAPER.md L176).  Written as CSV rows into the JSON and to <out>.profile.csv.
  placement  BASELINE.json configs[4]: 256 experts onto 8 virtual GPUs with throughput scales
             U[0.78,1.0]; loads = routing histograms (vibe_route_topk) for Zipf s in
             {0.8,1.2,1.6} x T in {2K,16K,64K}; contiguous vs token-balanced vs latency-balanced
             (ViBE Alg. 1 phase 2) under the measured C3-shape profile, model kinds A and B,
             cap = 32 and cap = 0.
  variability    1000 consecutive executions at 4K tokens per expert on this device: time per
                 execution from a cold start into the power-capped steady state, SM clock and power alongside.
  rack           rack-scale projection: the three policies for G = 8..128 virtual GPUs.
  recalibration  drift monitor + Algorithm 2 on a routing distribution that drifts: when it fires, how many
                 swaps repair the placement versus how many experts a full re-solve moves.

Everything here calls the CUDA library; nothing imports oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np
import torch

from . import binding as B
from . import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "kind": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "kind": "fallback"}


def _time(fn, iters, warmup=5, period=1):
    """Average CUDA-event time [us] of one fn(i) call.  `period` consecutive calls (one per
    rotating buffer set) are captured into a CUDA graph and the graph is replayed, so the
    number is the device time of the kernels, not the host's launch rate."""
    for i in range(max(warmup, period)):
        fn(i)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for i in range(period):
            fn(i)
    reps = max(1, iters // period)
    g.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e3 / (reps * period)


_FLUSH = None


def _time_cold(fn, iters, warmup=3):
    """Median CUDA-event time [us] of one fn() call that starts with a FLUSHED L2 (vibe_l2_flush before every timed
    call, outside the event pair): what a kernel costs inside a model, where other layers have evicted its operands.
    The call is captured into a CUDA graph, so the events bracket device time only."""
    global _FLUSH
    if _FLUSH is None:
        _FLUSH = torch.zeros((256 << 20,), dtype=torch.uint8, device="cuda")
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    for a, b in ev:
        B.l2_flush(_FLUSH)
        a.record()
        g.replay()
        b.record()
    torch.cuda.synchronize()
    return float(np.median([a.elapsed_time(b) for a, b in ev])) * 1e3


def _dev_bf16(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


STRESS = I.LayerConfig("S64K-stress", T=65536, d=2048, f=768, E=256, k=8, E_loc=256, zipf_s=1.0)


def section_stages(peaks, quick, only=None):
    """a1/a3/a5 in isolation, cold buffers."""
    out = []
    hbm = peaks["hbm_gbs"]
    for cfg in (I.C1, I.C2, I.C3, STRESS):
        if only and cfg.name.split("-")[0] not in only:
            continue
        T, k, E, E_loc, d = cfg.T, cfg.k, cfg.E, cfg.E_loc, cfg.d
        A = T * k
        Rcap = B.rows_cap(T, k, E_loc, 1)
        per_set = T * E * 4 + T * d * 2 + 2 * Rcap * d * 2 + T * d * 2
        nsets = max(2, min(8, int(np.ceil(400e6 / per_set))))
        emap_np = I.make_expert_map(cfg, "contiguous", 0)
        emap = torch.from_numpy(emap_np).cuda() if E_loc < E else None
        bias = torch.from_numpy(I.make_select_bias(E, 0)).cuda() if cfg.has_select_bias else None
        rc = B.RouteConfig(select_bias=bias, **I.route_kwargs(cfg))
        sets = []
        for i in range(nsets):
            lg = torch.from_numpy(I.make_logits(T, E, cfg.zipf_s, i, cfg.alpha)).cuda()
            X = torch.randn((T, d), device="cuda", dtype=torch.float32).to(torch.bfloat16)
            s = {"lg": lg, "X": X,
                 "ids": torch.empty((T, k), dtype=torch.int32, device="cuda"),
                 "w": torch.empty((T, k), dtype=torch.float32, device="cuda"),
                 "counts": torch.empty((E,), dtype=torch.int32, device="cuda"),
                 "Xp": torch.empty((Rcap, d), dtype=torch.bfloat16, device="cuda"),
                 "Y": torch.randn((Rcap, d), device="cuda", dtype=torch.float32).to(torch.bfloat16)
                 if Rcap * d < 2 ** 31 else torch.zeros((Rcap, d), dtype=torch.bfloat16, device="cuda"),
                 "off": torch.empty((E_loc + 1,), dtype=torch.int32, device="cuda"),
                 "r2a": torch.empty((Rcap,), dtype=torch.int32, device="cuda"),
                 "a2r": torch.empty((A,), dtype=torch.int32, device="cuda"),
                 "out": torch.empty((T, d), dtype=torch.bfloat16, device="cuda")}
            sets.append(s)
        ws = torch.empty((max(16, B.workspace_bytes(B.WS_PERMUTE, T, k, E, E_loc, d, 0)),), dtype=torch.uint8,
                         device="cuda")

        def route(i):
            s = sets[i % nsets]
            B.route_topk(s["lg"], rc, out=(s["ids"], s["w"], s["counts"]))

        def permute(i):
            s = sets[i % nsets]
            B.permute(s["X"], s["ids"], s["counts"], emap, E, E_loc, 1, out=(s["Xp"], s["off"], s["r2a"], s["a2r"]),
                      ws=ws)

        def combine(i):
            s = sets[i % nsets]
            B.combine(s["Y"], s["a2r"], s["w"], T, k, out=s["out"])

        iters = 40 if quick else 200
        n0 = B.launch_count()
        route(0)
        l_route = B.launch_count() - n0
        n0 = B.launch_count()
        permute(0)
        l_perm = B.launch_count() - n0
        t_route = _time(route, iters, period=nsets)
        t_perm = _time(permute, iters, period=nsets)
        t_comb = _time(combine, iters, period=nsets)
        # the floor of the route OP on this box: a selection-free kernel that only streams the same logits once
        # (vibe_l2_flush: 16-byte loads, no arithmetic) -- what reading 4*T*E bytes costs including the launch
        lgb = [x["lg"].view(torch.uint8).view(-1) for x in sets]
        t_read = _time(lambda i: B.l2_flush(lgb[i % nsets]), iters, period=nsets)
        s0 = sets[0]
        R = int(s0["off"][-1].item())
        res_tok = int((s0["a2r"].view(T, k) >= 0).any(dim=1).sum().item())
        by = {"route": 4.0 * T * E + 8.0 * T * k + 4.0 * E,
              "permute": 2.0 * res_tok * d + 2.0 * R * d + 12.0 * A,
              "combine": 2.0 * R * d + 2.0 * T * d + 8.0 * A}
        row = {"config": cfg.name, "T": T, "E": E, "E_loc": E_loc, "k": k, "d": d, "real_rows": R,
               "resident_tokens": res_tok, "buffer_sets": nsets, "set_bytes": per_set,
               "launches": {"route": l_route, "permute": l_perm, "combine": 1}}
        for name, t in (("route", t_route), ("permute", t_perm), ("combine", t_comb)):
            gbs = by[name] / t / 1e3
            row[name] = {"us": round(t, 2), "bytes": by[name], "GB/s": round(gbs, 1), "frac_hbm": round(gbs / hbm, 4),
                         "us_at_hbm_peak": round(by[name] / hbm / 1e3, 2)}
        row["route"]["logit_read_stream_us"] = round(t_read, 2)
        row["route"]["frac_of_read_stream"] = round(t_read / t_route, 4)
        out.append(row)
        del sets
        torch.cuda.empty_cache()
    return out


def section_fused(peaks, quick):
    """a4+a5: vibe_grouped_ffn + vibe_combine versus vibe_grouped_ffn_scatter + vibe_combine_scattered
    (gate-weighted scatter fused into the down projection) on the routed C1 / C2 batches."""
    out = []
    for cfg in (I.C1, I.C2):
        T, k, E, d, f = cfg.T, cfg.k, cfg.E, cfg.d, cfg.f
        W1, W3, W2 = _weights(E, d, f)
        rc = B.RouteConfig(**I.route_kwargs(cfg))
        lg = torch.from_numpy(I.make_logits(T, E, cfg.zipf_s, 0, cfg.alpha)).cuda()
        X = torch.randn((T, d), device="cuda").to(torch.bfloat16)
        ids, w, counts = B.route_topk(lg, rc)
        Xp, off, r2a, a2r = B.permute(X, ids, counts, None, E, E, 1)
        H = torch.empty((Xp.shape[0], f), dtype=torch.bfloat16, device="cuda")
        Y = torch.empty_like(Xp)
        Yw = torch.empty((T * k, d), dtype=torch.bfloat16, device="cuda")
        o = torch.empty((T, d), dtype=torch.bfloat16, device="cuda")

        def plain(i):
            B.grouped_ffn(Xp, off, W1, W3, W2, H=H, Y=Y)
            B.combine(Y, a2r, w, T, k, out=o)

        def fused(i):
            B.grouped_ffn_scatter(Xp, off, W1, W3, W2, r2a, w, H=H, Yw=Yw)
            B.combine_scattered(Yw, a2r, T, k, out=o)

        t0 = time.time()
        while time.time() - t0 < (0.3 if quick else 1.5):
            plain(0)
            torch.cuda.synchronize()
        iters = 20 if quick else 100
        tp = _time(plain, iters)
        tf = _time(fused, iters)
        out.append({"config": cfg.name, "ffn_plus_combine_us": round(tp, 2), "fused_scatter_us": round(tf, 2),
                    "speedup": round(tp / tf, 4)})
        del W1, W3, W2
        torch.cuda.empty_cache()
    return out


def section_layer(peaks, quick):
    """The whole layer (route -> permute -> grouped FFN -> combine) through vibe_moe_layer_forward: eager
    launches (6 kernels + 1 memset enqueued by one C call) versus the same call captured in a CUDA graph."""
    out = []
    for cfg in (I.C1, I.C2, I.C3):
        T, k, E, E_loc, d, f = cfg.T, cfg.k, cfg.E, cfg.E_loc, cfg.d, cfg.f
        W1, W3, W2 = _weights(E_loc, d, f)
        emap = torch.from_numpy(I.make_expert_map(cfg, "contiguous", 0)).cuda() if E_loc < E else None
        bias = torch.from_numpy(I.make_select_bias(E, 0)).cuda() if cfg.has_select_bias else None
        rc = B.RouteConfig(select_bias=bias, **I.route_kwargs(cfg))
        nsets = 4
        lgs = [torch.from_numpy(I.make_logits(T, E, cfg.zipf_s, i, cfg.alpha)).cuda() for i in range(nsets)]
        Xs = [torch.randn((T, d), device="cuda").to(torch.bfloat16) for _ in range(nsets)]
        o = torch.empty((T, d), dtype=torch.bfloat16, device="cuda")
        cnt = torch.empty((E,), dtype=torch.int32, device="cuda")
        arena = torch.empty((B.workspace_bytes(B.WS_LAYER, T, k, E, E_loc, d, f),), dtype=torch.uint8, device="cuda")

        def layer(i):
            B.moe_layer_forward(rc, lgs[i % nsets], Xs[i % nsets], emap, W1, W3, W2, out=o, counts=cnt, arena=arena)

        t0 = time.time()
        while time.time() - t0 < (0.3 if quick else 1.5):
            for i in range(8):
                layer(i)
            torch.cuda.synchronize()
        iters = 40 if quick else 200
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(iters):
            layer(i)
        e1.record()
        torch.cuda.synchronize()
        eager = e0.elapsed_time(e1) * 1e3 / iters
        graph = _time(layer, iters, period=nsets)
        row = {"config": cfg.name, "eager_us": round(eager, 1), "graph_us": round(graph, 1),
               "tokens_per_s_eager": round(T / eager * 1e6), "tokens_per_s_graph": round(T / graph * 1e6)}
        # the same layer with the FP8 FFN (weights packed once, outside the timed region)
        W1q, s1 = B.fp8_pack_weights(W1)
        W3q, s3 = B.fp8_pack_weights(W3)
        W2q, s2 = B.fp8_pack_weights(W2)
        hs = torch.full((E_loc,), 8.0 / 448.0, dtype=torch.float32, device="cuda")
        arena8 = torch.empty((B.workspace_bytes(B.WS_LAYER_FP8, T, k, E, E_loc, d, f),), dtype=torch.uint8, device="cuda")

        def layer8(i):
            B.moe_layer_forward_fp8(rc, lgs[i % nsets], Xs[i % nsets], emap, W1q, s1, W3q, s3, W2q, s2, hs, out=o,
                                    counts=cnt, arena=arena8)

        for i in range(8):
            layer8(i)
        torch.cuda.synchronize()
        g8 = _time(layer8, iters, period=nsets)
        row.update({"fp8_graph_us": round(g8, 1), "fp8_tokens_per_s_graph": round(T / g8 * 1e6),
                    "fp8_speedup": round(graph / g8, 3)})
        out.append(row)
        del W1, W3, W2, Xs, lgs, arena, W1q, W3q, W2q, arena8
        torch.cuda.empty_cache()
    return out


def section_ffn_fp8(peaks, quick):
    """f2: vibe_grouped_ffn_fp8 on BALANCED routing (every expert n rows) for the C1/C2/C3 shapes, next to the
    bf16 kernel on the same box in the same run.  FP8 tensor peak = 2 x the measured bf16 peaks (the guide's
    nominal ratio, as the task's roofline rule prescribes for a dtype without its own measured peak)."""
    out = []
    for cfg in (I.C1, I.C2, I.C3):
        E, d, f = cfg.E_loc, cfg.d, cfg.f
        W1, W3, W2 = _weights(E, d, f)
        W1q, s1 = B.fp8_pack_weights(W1)
        W3q, s3 = B.fp8_pack_weights(W3)
        W2q, s2 = B.fp8_pack_weights(W2)
        hs = torch.full((E,), 8.0 / 448.0, dtype=torch.float32, device="cuda")
        # the block-scaled variant (readings Q5-Q8): same weights, one UE8M0 scale per row and 32 K elements
        W1m, sf13 = B.mxfp8_pack_weights(W1, B.MX_ROLE_GATE)
        W3m, sf13 = B.mxfp8_pack_weights(W3, B.MX_ROLE_UP, sf=sf13)
        W2m, sf2 = B.mxfp8_pack_weights(W2, B.MX_ROLE_DOWN)
        for n in ((512, 2048) if quick else (128, 512, 1024, 2048, 4096)):
            R = E * n
            Xp = torch.randn((R, d), device="cuda").to(torch.bfloat16)
            Xq, rs = B.fp8_quantize_rows(Xp)
            off = (torch.arange(E + 1, device="cuda", dtype=torch.int32) * n).contiguous()
            Hq = torch.empty((R, f), dtype=torch.uint8, device="cuda")
            H = torch.empty((R, f), dtype=torch.bfloat16, device="cuda")
            Y = torch.empty((R, d), dtype=torch.bfloat16, device="cuda")
            f8 = lambda i: B.grouped_ffn_fp8(Xq, rs, off, W1q, s1, W3q, s3, W2q, s2, hs, Hq=Hq, Y=Y)
            Xm, xsf = B.mxfp8_quantize_rows(Xp, 32, B.MX_SF_TOKENS, R_cap=R)     # n is a multiple of 64: offsets aligned
            hsf = torch.full((max(16, B.mxfp8_sf_bytes(B.MX_SF_TOKENS, R, f)),), 127, dtype=torch.uint8, device="cuda")
            mx = lambda i: B.grouped_ffn_mxfp8(Xm, xsf, off, W1m, W3m, sf13, W2m, sf2, Hq=Hq, Hsf=hsf, Y=Y)
            bf = lambda i: B.grouped_ffn(Xp, off, W1, W3, W2, H=H, Y=Y)
            t0 = time.time()
            while time.time() - t0 < (0.2 if quick else 1.0):
                f8(0)
                torch.cuda.synchronize()
            iters = 20 if quick else 60
            t8 = _time(f8, iters)
            tb = _time(bf, iters)
            tq = _time(lambda i: B.fp8_quantize_rows(Xp), iters)
            tm = _time(mx, iters)
            tmq = _time(lambda i: B.mxfp8_quantize_rows(Xp, 32, B.MX_SF_TOKENS, R_cap=R), iters)
            flops = 6.0 * R * d * f
            out.append({"shape": cfg.name, "tokens_per_expert": n, "fp8_us": round(t8, 1), "bf16_us": round(tb, 1),
                        "quantize_rows_us": round(tq, 1), "fp8_TFLOP/s": round(flops / t8 / 1e6, 1),
                        "bf16_TFLOP/s": round(flops / tb / 1e6, 1), "speedup": round(tb / t8, 3),
                        "fp8_frac_of_2x_bf16_sustained": round(flops / t8 / 1e6 / (2 * peaks["bf16_tflops_sustained"]), 4),
                        "fp8_frac_of_2x_bf16_burst": round(flops / t8 / 1e6 / (2 * peaks["bf16_tflops"]), 4),
                        "mxfp8_us": round(tm, 1), "mxfp8_quantize_rows_us": round(tmq, 1),
                        "mxfp8_TFLOP/s": round(flops / tm / 1e6, 1), "mxfp8_speedup_vs_bf16": round(tb / tm, 3),
                        "mxfp8_frac_of_2x_bf16_sustained": round(flops / tm / 1e6 / (2 * peaks["bf16_tflops_sustained"]), 4),
                        "mxfp8_frac_of_2x_bf16_burst": round(flops / tm / 1e6 / (2 * peaks["bf16_tflops"]), 4)})
            del Xp, Xq, Hq, H, Y, Xm, xsf, hsf
        del W1, W3, W2, W1q, W3q, W2q, W1m, W3m, W2m, sf13, sf2
        torch.cuda.empty_cache()
    return out


def section_fp8_probe(peaks, quick):
    """A fixed, short launch sequence for ncu captures of the two FP8 kinds: C1 shape, 8 experts x 1024 rows; three
    calls of the block-scaled FFN, then three of the per-tensor one (launches 1-6 and 7-12 of ffn_gemm_kernel)."""
    cfg = I.C1
    E, d, f, n = cfg.E_loc, cfg.d, cfg.f, 1024
    W1, W3, W2 = _weights(E, d, f)
    R = E * n
    Xp = torch.randn((R, d), device="cuda").to(torch.bfloat16)
    off = (torch.arange(E + 1, device="cuda", dtype=torch.int32) * n).contiguous()
    W1m, sf13 = B.mxfp8_pack_weights(W1, B.MX_ROLE_GATE)
    W3m, sf13 = B.mxfp8_pack_weights(W3, B.MX_ROLE_UP, sf=sf13)
    W2m, sf2 = B.mxfp8_pack_weights(W2, B.MX_ROLE_DOWN)
    Xm, xsf = B.mxfp8_quantize_rows(Xp, 32, B.MX_SF_TOKENS, R_cap=R)
    for _ in range(3):
        B.grouped_ffn_mxfp8(Xm, xsf, off, W1m, W3m, sf13, W2m, sf2)
    torch.cuda.synchronize()
    del W1m, W3m, W2m
    (W1q, s1), (W3q, s3), (W2q, s2) = (B.fp8_pack_weights(w) for w in (W1, W3, W2))
    Xq, rs = B.fp8_quantize_rows(Xp)
    hs = torch.full((E,), 8.0 / 448.0, dtype=torch.float32, device="cuda")
    for _ in range(3):
        B.grouped_ffn_fp8(Xq, rs, off, W1q, s1, W3q, s3, W2q, s2, hs)
    torch.cuda.synchronize()
    return {"shape": cfg.name, "rows_per_expert": n, "calls": "3 x vibe_grouped_ffn_mxfp8, then 3 x vibe_grouped_ffn_fp8"}


def _weights(E, d, f):
    W1 = (torch.randn((E, d, f), device="cuda") * d ** -0.5).to(torch.bfloat16)
    W3 = (torch.randn((E, d, f), device="cuda") * d ** -0.5).to(torch.bfloat16)
    W2 = (torch.randn((E, f, d), device="cuda") * f ** -0.5).to(torch.bfloat16)
    return W1, W3, W2


def _warm(W1, W3, W2, seconds=2.0):
    """'Each GPU is warmed to steady-state operating conditions': back-to-back
    grouped FFN at 1024 tokens per expert for `seconds`."""
    t0 = time.time()
    while time.time() - t0 < seconds:
        B.profile_expert_latency(W1, W3, W2, (1024,), mode=0, warmup=0, iters=20)


def section_ffn(peaks, quick):
    out = []
    sweep = (128, 256, 512, 1024, 2048, 4096)
    for cfg in (I.C1, I.C2, I.C3):
        E, d, f = cfg.E_loc, cfg.d, cfg.f
        W1, W3, W2 = _weights(E, d, f)
        _warm(W1, W3, W2, 0.5 if quick else 2.0)
        # largest point first: the sweep starts in the power-capped steady state the warm loop left, and
        # every point gets enough untimed calls to ride out the DVFS transient of a change in intensity
        lat = B.profile_expert_latency(W1, W3, W2, sweep[::-1], mode=0, warmup=10 if quick else 30,
                                       iters=20 if quick else 50)[::-1]
        for n, l in zip(sweep, lat):
            tf = 6.0 * n * d * f / l / 1e6
            bytes_e = 6.0 * d * f + 4.0 * n * d + 4.0 * n * f
            t_roof = max(6.0 * n * d * f / (peaks["bf16_tflops_sustained"] * 1e6), bytes_e / (peaks["hbm_gbs"] * 1e3))
            out.append({"shape": cfg.name, "E_loc": E, "d": d, "f": f, "tokens_per_expert": n,
                        "us_per_expert": round(float(l), 3), "TFLOP/s": round(tf, 1),
                        "frac_sustained": round(tf / peaks["bf16_tflops_sustained"], 4),
                        "frac_burst": round(tf / peaks["bf16_tflops"], 4),
                        "frac_of_per_expert_roofline": round(t_roof / float(l), 4)})
        del W1, W3, W2
        torch.cuda.empty_cache()
    return out


def section_mixed(peaks, quick):
    """Grouped FFN on skewed row distributions (S8(f) f4): a lone light expert, a few light
    experts, every expert light, and heavy experts mixed with light ones.  The first case runs first with a fixed
    number of launches, so that an ncu capture of the first ffn_gemm_kernel launches is the lone expert."""
    out = []
    cases = [("C3", I.C3, "1 x 32", [32] + [0] * 31), ("C3", I.C3, "4 x 32", [32] * 4 + [0] * 28),
             ("C3", I.C3, "32 x 32", [32] * 32), ("C3", I.C3, "4 x 2048", [2048] * 4 + [0] * 28),
             ("C3", I.C3, "4 x 2048 + 28 x 32", [2048] * 4 + [32] * 28),
             ("C3", I.C3, "8 x 1024 + 24 x 64", [1024] * 8 + [64] * 24),
             ("C2", I.C2, "128 x 16", [16] * 128), ("C2", I.C2, "24 x 1024", [1024] * 24 + [0] * 104),
             ("C2", I.C2, "24 x 1024 + 104 x 64", [1024] * 24 + [64] * 104)]
    held = {}
    fws = torch.empty((max(16, B.workspace_bytes(B.WS_FFN, 1, 1, 1, 1, 64, 64)),), dtype=torch.uint8, device="cuda")
    warmed = False
    for shape, cfg, label, rows in cases:
        E, d, f = cfg.E_loc, cfg.d, cfg.f
        if shape not in held:
            held.clear()
            torch.cuda.empty_cache()
            held[shape] = _weights(E, d, f)
        W1, W3, W2 = held[shape]
        R = int(sum(rows))
        Xp = torch.randn((R, d), device="cuda").to(torch.bfloat16)
        H = torch.empty((R, f), dtype=torch.bfloat16, device="cuda")
        Y = torch.empty((R, d), dtype=torch.bfloat16, device="cuda")
        off = torch.tensor(np.concatenate([[0], np.cumsum(rows)]), dtype=torch.int32, device="cuda")
        if not warmed:          # the first case must not be timed on a device that is still ramping its clocks
            t0 = time.time()
            while time.time() - t0 < (0.3 if quick else 1.0):
                B.grouped_ffn(Xp, off, W1, W3, W2, H, Y, ws=fws)
                torch.cuda.synchronize()
            warmed = True
        # timed twice, the smaller kept: the first case follows an idle device (weights just generated).
        # `us` = back-to-back replays (operands that fit the 126 MB L2 stay there: a lone C3 expert has 88 MB of
        # weights); `cold_us` = every call after an L2 flush; `no_split_cold_us` = the same without the split-K workspace
        us = min(_time(lambda i: B.grouped_ffn(Xp, off, W1, W3, W2, H, Y, ws=fws), 20 if quick else 100, warmup=3)
                 for _ in range(2))
        cold = _time_cold(lambda: B.grouped_ffn(Xp, off, W1, W3, W2, H, Y, ws=fws), 15 if quick else 41)
        cold_ns = _time_cold(lambda: B.grouped_ffn(Xp, off, W1, W3, W2, H, Y, ws=None), 15 if quick else 41)
        active = sum(1 for r in rows if r > 0)
        floor_us = (active * 6.0 * d * f + 4.0 * R * d + 4.0 * R * f) / (peaks["hbm_gbs"] * 1e3)
        out.append({"shape": shape, "rows_per_expert": label, "rows": R, "active_experts": active, "us": round(us, 1),
                    "cold_us": round(cold, 1), "no_split_cold_us": round(cold_ns, 1),
                    "weight_stream_floor_us": round(floor_us, 1), "cold_over_floor": round(cold / floor_us, 2),
                    "weight_TB/s": round(active * 6.0 * d * f / us / 1e6, 2),
                    "cold_weight_TB/s": round(active * 6.0 * d * f / cold / 1e6, 2),
                    "TFLOP/s": round(6.0 * R * d * f / us / 1e6, 1)})
    return out


def section_profile(peaks, quick):
    out = {}
    for cfg in (I.C2, I.C3):
        E, d, f = cfg.E_loc, cfg.d, cfg.f
        W1, W3, W2 = _weights(E, d, f)
        _warm(W1, W3, W2, 0.5 if quick else 2.0)
        rows = []
        for mode in (0, 1):
            lat, samples = B.profile_expert_latency(W1, W3, W2, B.DEFAULT_SWEEP[::-1], mode=mode,
                                                    warmup=10 if quick else 30, iters=20 if quick else 100,
                                                    return_samples=True)
            lat, samples = lat[::-1], samples[::-1]      # measured from the largest point down (steady state)
            if mode == 0:
                samples = samples / E
            for j, n in enumerate(B.DEFAULT_SWEEP):
                floor_us = 6.0 * d * f / (peaks["hbm_gbs"] * 1e3)      # the expert's weight bytes at HBM peak
                rows.append({"mode": mode, "tokens_per_expert": int(n), "latency_us": round(float(lat[j]), 3),
                             "p10_us": round(float(np.percentile(samples[j], 10)), 3),
                             "p90_us": round(float(np.percentile(samples[j], 90)), 3),
                             "weight_stream_floor_us": round(floor_us, 3) if mode == 0 else None})
        # the same sweep for the FP8 FFN (mode 0): the per-GPU performance model in the paper's precision
        W1q, s1 = B.fp8_pack_weights(W1)
        W3q, s3 = B.fp8_pack_weights(W3)
        W2q, s2 = B.fp8_pack_weights(W2)
        hs = torch.full((E,), 8.0 / 448.0, dtype=torch.float32, device="cuda")
        lat8 = B.profile_expert_latency_fp8(W1q, s1, W3q, s3, W2q, s2, hs, B.DEFAULT_SWEEP[::-1], mode=0,
                                            warmup=10 if quick else 30, iters=20 if quick else 100)[::-1]
        m0 = [r for r in rows if r["mode"] == 0]
        for j, r in enumerate(m0):
            r["fp8_latency_us"] = round(float(lat8[j]), 3)
        del W1q, W3q, W2q
        # ... and for the BLOCK-SCALED FP8 FFN (segments padded to 64 rows: l(n) is a step function of n)
        W1m, sf13 = B.mxfp8_pack_weights(W1, B.MX_ROLE_GATE)
        W3m, sf13 = B.mxfp8_pack_weights(W3, B.MX_ROLE_UP, sf=sf13)
        W2m, sf2 = B.mxfp8_pack_weights(W2, B.MX_ROLE_DOWN)
        latm = B.profile_expert_latency_mxfp8(W1m, W3m, sf13, W2m, sf2, B.DEFAULT_SWEEP[::-1], mode=0,
                                              warmup=10 if quick else 30, iters=20 if quick else 100)[::-1]
        for j, r in enumerate(m0):
            r["mxfp8_latency_us"] = round(float(latm[j]), 3)
        del W1m, W3m, W2m
        out[cfg.name] = {"E_loc": E, "d": d, "f": f, "rows": rows}
        del W1, W3, W2
        torch.cuda.empty_cache()
    return out


def section_placement(peaks, quick, profile):
    """BASELINE.json configs[4] on the measured C3-shape profile (mode 0)."""
    model, _ = _c3_model(peaks, profile)
    E, G, k = 256, 8, 8
    rc = B.RouteConfig(num_experts=E, top_k=k)
    out = []
    for s in (0.8, 1.2, 1.6):
        for T in (2048, 16384, 65536):
            lg = torch.from_numpy(I.make_logits(T, E, s, 7, 1.0)).cuda()
            _, _, counts = B.route_topk(lg, rc)
            load = counts.cpu().numpy().astype(np.float64)
            for seed in range(2 if quick else 8):
                scale = I.make_throughput_scales(G, seed)
                for cap in (E // G, 0):
                    binnings = {"contiguous": B.placement_contiguous(E, G),
                                "token_balanced": B.placement_token_balanced(load, G, cap),
                                "latency_balanced": B.placement_greedy(load, G, scale, model, cap)}
                    for kind, kname in ((B.MODEL_A, "A"), (B.MODEL_B, "B")):
                        row = {"zipf_s": s, "T": T, "scale_seed": seed, "cap": cap, "model": kname}
                        for name, asg in binnings.items():
                            sc, per = B.placement_eval(asg, load, G, scale, model, kind)
                            row[name] = {"score_us": round(sc, 3), "max_over_mean": round(sc / float(per.mean()), 4)}
                        row["gain_latency_vs_token"] = round(1.0 - row["latency_balanced"]["score_us"] /
                                                             row["token_balanced"]["score_us"], 4)
                        row["gain_latency_vs_contiguous"] = round(1.0 - row["latency_balanced"]["score_us"] /
                                                                  row["contiguous"]["score_us"], 4)
                        out.append(row)
    return out


def _c3_model(peaks, profile):
    if profile is None:
        profile = section_profile(peaks, True)
    prof = [r for r in profile[I.C3.name]["rows"] if r["mode"] == 0]
    return B.LatencyModel([r["tokens_per_expert"] for r in prof], [r["latency_us"] for r in prof],
                          E_prof=profile[I.C3.name]["E_loc"]), profile


def section_variability(peaks, quick):
    """The paper's variability protocol on THIS device: "4K tokens per expert ... 1000 consecutive MoE
    layer executions" under perfect balance, C3 shape: per-execution kernel time and the
    SM clock over the run -- how much one GPU's own DVFS moves f(n) between a cold start and steady state."""
    cfg = I.C3
    E, d, f = cfg.E_loc, cfg.d, cfg.f
    W1, W3, W2 = _weights(E, d, f)
    n_exec = 200 if quick else 1000
    clocks, power = [], []
    try:
        import pynvml
        import threading
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(torch.cuda.current_device())
        stop = threading.Event()

        def sample():
            while not stop.is_set():
                clocks.append(int(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
                time.sleep(0.01)
        th = threading.Thread(target=sample, daemon=True)
        th.start()
    except Exception:
        stop, th = None, None
    time.sleep(1.0)                                  # let the device idle: the run starts cold
    lat, samples = B.profile_expert_latency(W1, W3, W2, (4096,), mode=0, warmup=0, iters=n_exec, return_samples=True)
    if stop is not None:
        stop.set()
        th.join(timeout=2)
    t = samples[0]                                   # whole-kernel time per execution [us]
    flops = 6.0 * E * 4096 * d * f
    q = lambda a, p: float(np.percentile(a, p))
    out = {"shape": cfg.name, "tokens_per_expert": 4096, "executions": n_exec,
           "us_first_10": round(float(t[:10].mean()), 1), "us_last_100": round(float(t[-100:].mean()), 1),
           "us_median": round(q(t, 50), 1), "us_p1": round(q(t, 1), 1), "us_p99": round(q(t, 99), 1),
           "slowdown_steady_vs_cold": round(float(t[-100:].mean() / t[:10].mean()), 4),
           "spread_p99_over_p1": round(q(t, 99) / q(t, 1), 4),
           "tflops_first_10": round(flops / float(t[:10].mean()) / 1e6, 1),
           "tflops_last_100": round(flops / float(t[-100:].mean()) / 1e6, 1),
           "sm_mhz_max": max(clocks) if clocks else None, "sm_mhz_min_under_load": min(clocks) if clocks else None,
           "sm_mhz_last": clocks[-1] if clocks else None, "power_w_max": round(max(power), 1) if power else None}
    del W1, W3, W2
    torch.cuda.empty_cache()
    return out


def section_rack(peaks, quick, profile):
    """Rack-scale projection (Fig. 15): the same three policies as G grows
    from 8 to 128 virtual GPUs, sigma_g resampled per G, equal experts per GPU (cap = E/G), model B."""
    model, _ = _c3_model(peaks, profile)
    E, k = 256, 8
    rc = B.RouteConfig(num_experts=E, top_k=k)
    lg = torch.from_numpy(I.make_logits(16384, E, 1.2, 7, 1.0)).cuda()
    load = B.route_topk(lg, rc)[2].cpu().numpy().astype(np.float64)
    return rack_sweep(load, model, E, (8, 16, 32, 64, 128), range(4 if quick else 16))


def rack_sweep(load, model, E, Gs, seeds):
    """The evaluator sweep behind the rack-scale projection (host only: placement calls of the C ABI): for every G,
    sigma_g resampled per seed (inputs.make_throughput_scales(G, 100 + seed)), cap = E/G, model B; gain of the
    latency-balanced greedy over the token-balanced one and over contiguous placement, and max/mean bin latency of
    the latency-balanced placement.  tests/test_report_host.py pins it against the oracle's placement functions."""
    out = []
    for G in Gs:
        gains_t, gains_c, ratio = [], [], []
        for seed in seeds:
            scale = I.make_throughput_scales(G, 100 + seed)
            cap = E // G
            tb = B.placement_token_balanced(load, G, cap)
            lb = B.placement_greedy(load, G, scale, model, cap)
            ct = B.placement_contiguous(E, G)
            s_tb = B.placement_eval(tb, load, G, scale, model, B.MODEL_B)[0]
            s_lb, per = B.placement_eval(lb, load, G, scale, model, B.MODEL_B)
            s_ct = B.placement_eval(ct, load, G, scale, model, B.MODEL_B)[0]
            gains_t.append(1.0 - s_lb / s_tb)
            gains_c.append(1.0 - s_lb / s_ct)
            ratio.append(s_lb / float(per.mean()))
        out.append({"G": G, "experts_per_gpu": E // G,
                    "gain_latency_vs_token_median": round(float(np.median(gains_t)), 4),
                    "gain_latency_vs_token_min": round(float(min(gains_t)), 4),
                    "gain_latency_vs_token_max": round(float(max(gains_t)), 4),
                    "gain_latency_vs_contiguous_median": round(float(np.median(gains_c)), 4),
                    "latency_balanced_max_over_mean_median": round(float(np.median(ratio)), 4)})
    return out


def section_recalibration(peaks, quick, profile):
    """Online recalibration (Alg. 1 phase 3 + Alg. 2): the routing distribution drifts from one Zipf
    permutation to another over 200 passes; the drift monitor (window 100, H 10, delta 0.05) fires, the swap
    solver repairs the stale latency-balanced placement; swaps applied versus experts a full re-solve moves."""
    model, _ = _c3_model(peaks, profile)
    E, G, k, T = 256, 8, 8, 4096
    rc = B.RouteConfig(num_experts=E, top_k=k)
    scale = I.make_throughput_scales(G, 3)
    base_a = torch.from_numpy(I.make_logits(T, E, 1.2, 21, 1.0)).cuda()
    bias_a = torch.from_numpy(I.zipf_bias(E, 1.2, 21)).cuda()
    bias_b = torch.from_numpy(I.zipf_bias(E, 1.2, 22)).cuda()
    mon = B.DriftMonitor(1, E, 100, 10, 0.05)
    events, assign, passes = [], None, 300 if quick else 600
    for p in range(1, passes + 1):
        mix = 0.0 if p <= 150 else min(1.0, (p - 150) / 200.0)
        lg = base_a - bias_a[None, :] + ((1 - mix) * bias_a + mix * bias_b)[None, :]
        load = B.route_topk(lg.contiguous(), rc)[2].cpu().numpy().astype(np.float64)
        trig, dist = mon.push(load[None, :])
        if p == 100:
            w = mon.window_mean()[0]
            mon.set_reference(w[None, :])
            assign = B.placement_greedy(w, G, scale, model, E // G)
        if trig:
            w = mon.window_mean()[0]
            before = B.placement_eval(assign, w, G, scale, model, B.MODEL_B)[0]
            fixed, swaps = B.placement_swap_refine(assign, w, G, scale, model, B.MODEL_B, 0.03)
            after = B.placement_eval(fixed, w, G, scale, model, B.MODEL_B)[0]
            full = B.placement_greedy(w, G, scale, model, E // G)
            events.append({"pass": p, "cosine_distance": round(float(dist[0]), 4), "swaps": len(swaps),
                           "experts_moved_by_swaps": int((fixed != assign).sum()),
                           "experts_moved_by_full_resolve": int((full != assign).sum()),
                           "score_before_us": round(before, 2), "score_after_swaps_us": round(after, 2),
                           "score_full_resolve_us": round(B.placement_eval(full, w, G, scale, model, B.MODEL_B)[0], 2)})
            assign = fixed
            mon.rearranged()
    mon.close()
    return {"passes": passes, "drift": "Zipf(1.2) expert permutation A -> B, linear over passes 150..350", "events": events}


def write_markdown(r, path, command):
    """The JSON report as markdown tables (what profiles/r1_report.md holds)."""
    import collections
    import statistics as st
    o=[]
    o.append("# per-kernel measurements on one B200 (`python -m paper_2606_00735_b200.report`)\n")
    o.append("Command (under gpurun, one B200, no profiler attached):\n\n    " + command + "\n")
    o.append(f"Peaks ({r['peaks']['kind']}, MEASURED_PEAKS.json): HBM copy {r['peaks']['hbm_gbs']} GB/s; cuBLAS bf16 {r['peaks']['bf16_tflops']} TFLOP/s burst, {r['peaks']['bf16_tflops_sustained']} sustained.  GPU: {r['gpu']}.\n")
    if "stages" in r:
        o.append("## stages: route / permute / combine, each timed alone from a CUDA graph over rotating cold buffer sets\n")
        o.append("achieved = algorithmic bytes (DESIGN.md section 7) / device time; `frac` = achieved / measured HBM copy peak.\n")
        o.append("| config | T | E (resident) | k | d | real rows | route us | GB/s | frac | logits read once (vibe_l2_flush) us | permute us | GB/s | frac | combine us | GB/s | frac |")
        o.append("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        for s in r['stages']:
            o.append(f"| {s['config']} | {s['T']} | {s['E']} ({s['E_loc']}) | {s['k']} | {s['d']} | {s['real_rows']} | "
                     f"{s['route']['us']} | {s['route']['GB/s']} | {s['route']['frac_hbm']} | {s['route'].get('logit_read_stream_us', '')} | "
                     + " | ".join(f"{s[n]['us']} | {s[n]['GB/s']} | {s[n]['frac_hbm']}" for n in ('permute', 'combine')) + " |")
        o.append("\nRoute: bound by the ALU pipe at 64K tokens and by launch + latency at the C1-C3 batch sizes, not by HBM (`r2_route_ncu.md`); the column beside it is the floor of the OP on this box: a selection-free kernel that only streams the same logits once.  permute = 2 launches (cooperative index kernel + row kernel), combine = 1.\n")
    if "ffn_balanced" in r:
        o.append("## ffn_balanced: grouped FFN, every expert n rows (vibe_profile_expert_latency mode 0, largest n first, 2 s warm loop)\n")
        o.append("| shape | E_loc | d | f | tokens/expert | us/expert | TFLOP/s | of sustained | of burst | of per-expert roofline max(flops/sustained, bytes/HBM) |")
        o.append("|---|---|---|---|---|---|---|---|---|---|")
        for x in r['ffn_balanced']:
            o.append(f"| {x['shape']} | {x['E_loc']} | {x['d']} | {x['f']} | {x['tokens_per_expert']} | {x['us_per_expert']} | {x['TFLOP/s']} | {x['frac_sustained']} | {x['frac_burst']} | {x['frac_of_per_expert_roofline']} |")
    if "ffn_mixed" in r:
        o.append("\n## ffn_mixed: grouped FFN on skewed row distributions (CUDA graph; weight TB/s = weights of the active experts / time)\n")
        o.append("| shape | rows per expert | rows | active experts | us (replayed) | weight TB/s | cold us (L2 flushed) | cold, no split-K | weight-stream floor us | cold / floor | TFLOP/s |")
        o.append("|---|---|---|---|---|---|---|---|---|---|---|")
        for x in r["ffn_mixed"]:
            o.append(f"| {x['shape']} | {x['rows_per_expert']} | {x['rows']} | {x['active_experts']} | {x['us']} | {x['weight_TB/s']} | {x.get('cold_us', '')} | {x.get('no_split_cold_us', '')} | {x.get('weight_stream_floor_us', '')} | {x.get('cold_over_floor', '')} | {x['TFLOP/s']} |")
        o.append("\nA light expert occupies its CTA pairs for (weight bytes of the tile) / ~140 GB/s whatever else runs (DESIGN.md section 12): heavy and light experts add; with at most half as many tiles as CTA pairs the split-K path spreads a tile's K range over several pairs.\n")
    if "fused_scatter" in r:
        o.append("\n## fused_scatter: vibe_grouped_ffn + vibe_combine vs vibe_grouped_ffn_scatter + vibe_combine_scattered (routed batches)\n")
        o.append("| config | ffn + combine us | fused scatter us | speedup |\n|---|---|---|---|")
        for x in r['fused_scatter']:
            o.append(f"| {x['config']} | {x['ffn_plus_combine_us']} | {x['fused_scatter_us']} | {x['speedup']} |")
    if "profile" in r:
        o.append("\n## profile: per-expert latency l(n) [us], median of 100 calls per point (p10..p90), modes 0 (all experts n rows; time / E_loc) and 1 (one expert n rows)\n")
        for name,p in r['profile'].items():
            o.append(f"### {name}: E_loc={p['E_loc']} d={p['d']} f={p['f']}\n")
            o.append("| n | mode 0 us | p10 | p90 | weight-stream floor us | mode 1 us | p10 | p90 | per-tensor FP8 mode 0 us | block-scaled FP8 mode 0 us |\n|---|---|---|---|---|---|---|---|---|---|")
            m0={x['tokens_per_expert']:x for x in p['rows'] if x['mode']==0}
            m1={x['tokens_per_expert']:x for x in p['rows'] if x['mode']==1}
            for n in sorted(m0):
                a,b=m0[n],m1[n]
                o.append(f"| {n} | {a['latency_us']} | {a['p10_us']} | {a['p90_us']} | {a['weight_stream_floor_us']} | {b['latency_us']} | {b['p10_us']} | {b['p90_us']} | {a.get('fp8_latency_us')} | {a.get('mxfp8_latency_us')} |")
            o.append("")
    if "placement_stress" in r:
        o.append("## placement_stress (BASELINE.json configs[4]): 256 experts -> 8 virtual GPUs, sigma ~ U[0.78,1.0] (8 seeds), measured C3-shape profile\n")
        o.append("score = max over bins of modelled latency / sigma [us]; gain = 1 - latency-balanced / token-balanced.  Medians over the 8 scale draws.\n")
        o.append("| zipf s | T | cap | model | contiguous | token-balanced | latency-balanced (ViBE) | gain vs token-balanced (median, min..max) | gain vs contiguous (median) |")
        o.append("|---|---|---|---|---|---|---|---|---|")
        g=collections.defaultdict(list)
        for x in r['placement_stress']: g[(x['zipf_s'],x['T'],x['cap'],x['model'])].append(x)
        for k_,v in sorted(g.items()):
            med=lambda f: round(st.median(f(y) for y in v),2)
            gt=[y['gain_latency_vs_token'] for y in v]
            o.append(f"| {k_[0]} | {k_[1]} | {k_[2]} | {k_[3]} | {med(lambda y:y['contiguous']['score_us'])} | {med(lambda y:y['token_balanced']['score_us'])} | {med(lambda y:y['latency_balanced']['score_us'])} | {round(st.median(gt),4)} ({min(gt)}..{max(gt)}) | {med(lambda y:y['gain_latency_vs_contiguous'])} |")
    if "ffn_fp8" in r:
        o.append("\n## ffn_fp8: the FP8 kinds of the grouped FFN vs vibe_grouped_ffn (bf16), balanced, same run: block-scaled e4m3 (vibe_grouped_ffn_mxfp8, UE8M0 scale per row and 32 K elements) and per-tensor e4m3 (vibe_grouped_ffn_fp8)\n")
        o.append("| shape | tokens/expert | bf16 us | bf16 TFLOP/s | block-scaled us | TFLOP/s | vs bf16 | of 2 x bf16 sustained | quantize rows us | per-tensor us | TFLOP/s | vs bf16 | of 2 x bf16 sustained | of 2 x bf16 burst | quantize rows us |")
        o.append("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        for x in r["ffn_fp8"]:
            o.append(f"| {x['shape']} | {x['tokens_per_expert']} | {x['bf16_us']} | {x['bf16_TFLOP/s']} | {x.get('mxfp8_us', '')} | {x.get('mxfp8_TFLOP/s', '')} | "
                     f"{x.get('mxfp8_speedup_vs_bf16', '')} | {x.get('mxfp8_frac_of_2x_bf16_sustained', '')} | {x.get('mxfp8_quantize_rows_us', '')} | "
                     f"{x['fp8_us']} | {x['fp8_TFLOP/s']} | {x['speedup']} | {x['fp8_frac_of_2x_bf16_sustained']} | {x['fp8_frac_of_2x_bf16_burst']} | {x['quantize_rows_us']} |")
    if "layer" in r:
        o.append("\n## layer: vibe_moe_layer_forward (route + permute + grouped FFN + combine), zipf-routed batches, 4 rotating input sets\n")
        o.append("| config | bf16 eager us | bf16 CUDA graph us | tokens/s eager | tokens/s graph | FP8 layer (vibe_moe_layer_forward_fp8) graph us | FP8 tokens/s | FP8 / bf16 |\n|---|---|---|---|---|---|---|---|")
        for x in r["layer"]:
            o.append(f"| {x['config']} | {x['eager_us']} | {x['graph_us']} | {x['tokens_per_s_eager']} | {x['tokens_per_s_graph']} | "
                     f"{x.get('fp8_graph_us')} | {x.get('fp8_tokens_per_s_graph')} | {x.get('fp8_speedup')} |")
    if "variability" in r:
        v = r["variability"]
        o.append("\n## variability: " + str(v["executions"]) + " consecutive executions, " + v["shape"] +
                 ", 4096 tokens per expert, from an idle device (PAPER.md L335 protocol)\n")
        o.append("| us first 10 | us last 100 | median | p1 | p99 | steady / cold | p99 / p1 | TFLOP/s first 10 | TFLOP/s last 100 | SM MHz max | min under load | last | power W max |")
        o.append("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        o.append("| " + " | ".join(str(v[k_]) for k_ in ("us_first_10", "us_last_100", "us_median", "us_p1", "us_p99",
                 "slowdown_steady_vs_cold", "spread_p99_over_p1", "tflops_first_10", "tflops_last_100", "sm_mhz_max",
                 "sm_mhz_min_under_load", "sm_mhz_last", "power_w_max")) + " |")
    if "rack_projection" in r:
        o.append("\n## rack_projection: 256 experts, Zipf 1.2, 16K tokens, sigma ~ U[0.78,1.0] resampled 16x per G, cap = E/G, model B\n")
        o.append("| G | experts/GPU | gain vs token-balanced: median | min | max | gain vs contiguous (median) | latency-balanced max/mean (median) |")
        o.append("|---|---|---|---|---|---|---|")
        for x in r["rack_projection"]:
            o.append(f"| {x['G']} | {x['experts_per_gpu']} | {x['gain_latency_vs_token_median']} | {x['gain_latency_vs_token_min']} | "
                     f"{x['gain_latency_vs_token_max']} | {x['gain_latency_vs_contiguous_median']} | {x['latency_balanced_max_over_mean_median']} |")
    if "recalibration" in r:
        c = r["recalibration"]
        o.append("\n## recalibration: drift monitor (window 100, H 10, delta 0.05) + Algorithm 2 (eps 0.03); " + c["drift"] + "\n")
        o.append("| pass | cosine distance | swaps | experts moved by swaps | moved by a full re-solve | score before us | after swaps | full re-solve |")
        o.append("|---|---|---|---|---|---|---|---|")
        for e in c["events"]:
            o.append(f"| {e['pass']} | {e['cosine_distance']} | {e['swaps']} | {e['experts_moved_by_swaps']} | "
                     f"{e['experts_moved_by_full_resolve']} | {e['score_before_us']} | {e['score_after_swaps_us']} | {e['score_full_resolve_us']} |")
    with open(path, "w") as fh:
        fh.write("\n".join(o) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sections", default="stages,ffn,mixed,fp8,fused,layer,profile,placement,variability,rack,recalibration")
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "report.json"))
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--md", default="", help="also write the report as markdown tables (needs all sections)")
    ap.add_argument("--configs", default="", help="stages section only: comma list out of C1,C2,C3,S64K")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("report: no CUDA device -- the product has no CPU fallback")
    B.load()
    torch.cuda.set_device(0)
    peaks = _peaks()
    rep = {"peaks": peaks, "gpu": torch.cuda.get_device_name(0)}
    want = args.sections.split(",")
    if "stages" in want:
        rep["stages"] = section_stages(peaks, args.quick, [c for c in args.configs.split(",") if c])
        for r in rep["stages"]:
            print(r["config"], {n: (r[n]["us"], r[n]["GB/s"], r[n]["frac_hbm"]) for n in ("route", "permute", "combine")},
                  flush=True)
    if "ffn" in want:
        rep["ffn_balanced"] = section_ffn(peaks, args.quick)
        for r in rep["ffn_balanced"]:
            print(r["shape"], r["tokens_per_expert"], r["us_per_expert"], r["TFLOP/s"], r["frac_sustained"], flush=True)
    if "mixed" in want:
        rep["ffn_mixed"] = section_mixed(peaks, args.quick)
        for r in rep["ffn_mixed"]:
            print(r, flush=True)
    if "fused" in want:
        rep["fused_scatter"] = section_fused(peaks, args.quick)
        for r in rep["fused_scatter"]:
            print(r, flush=True)
    if "fp8_probe" in want:
        rep["fp8_probe"] = section_fp8_probe(peaks, args.quick)
    if "fp8" in want:
        rep["ffn_fp8"] = section_ffn_fp8(peaks, args.quick)
        for r in rep["ffn_fp8"]:
            print(r, flush=True)
    if "layer" in want:
        rep["layer"] = section_layer(peaks, args.quick)
        for r in rep["layer"]:
            print(r, flush=True)
    if "profile" in want:
        rep["profile"] = section_profile(peaks, args.quick)
    if "placement" in want:
        rep["placement_stress"] = section_placement(peaks, args.quick, rep.get("profile"))
        g = [r["gain_latency_vs_token"] for r in rep["placement_stress"] if r["model"] == "B" and r["cap"] > 0]
        print(f"placement: latency- vs token-balanced gain (model B, cap 32): median {np.median(g):.3f} "
              f"min {min(g):.3f} max {max(g):.3f}", flush=True)
    if "variability" in want:
        rep["variability"] = section_variability(peaks, args.quick)
        print("variability", rep["variability"], flush=True)
    if "rack" in want:
        rep["rack_projection"] = section_rack(peaks, args.quick, rep.get("profile"))
        for r in rep["rack_projection"]:
            print("rack", r, flush=True)
    if "recalibration" in want:
        rep["recalibration"] = section_recalibration(peaks, args.quick, rep.get("profile"))
        for e in rep["recalibration"]["events"]:
            print("recalibration", e, flush=True)
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    with open(args.out, "w") as fh:
        json.dump(rep, fh, indent=1)
    if "profile" in rep:
        with open(args.out.replace(".json", "") + ".profile.csv", "w") as fh:
            fh.write("shape,mode,tokens_per_expert,latency_us,p10_us,p90_us,fp8_latency_us,mxfp8_latency_us\n")
            for name, p in rep["profile"].items():
                for r in p["rows"]:
                    fh.write(f"{name},{r['mode']},{r['tokens_per_expert']},{r['latency_us']},{r['p10_us']},{r['p90_us']},"
                             f"{r.get('fp8_latency_us', '')},{r.get('mxfp8_latency_us', '')}\n")
    if args.md:
        write_markdown(rep, args.md, "python -m paper_2606_00735_b200.report " + " ".join(sys.argv[1:]))
    print("wrote", args.out)


if __name__ == "__main__":
    sys.exit(main())
