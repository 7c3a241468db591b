"""CPU-only checks of the reporting helpers (no GPU work): the markdown writer accepts partial reports."""
import os

from paper_2606_00735_b200 import report


def test_write_markdown_with_partial_and_full_sections(tmp_path):
    rep = {"peaks": {"kind": "measured", "hbm_gbs": 6533.2, "bf16_tflops": 1665.5, "bf16_tflops_sustained": 1401.3},
           "gpu": "NVIDIA B200"}
    p = tmp_path / "a.md"
    report.write_markdown(rep, str(p), "cmd")
    assert "Peaks (measured" in p.read_text()
    stage = {"us": 1.0, "GB/s": 2.0, "frac_hbm": 0.5}
    rep.update({
        "stages": [{"config": "C1", "T": 1, "E": 8, "E_loc": 8, "k": 2, "d": 64, "real_rows": 2, "route": stage,
                    "permute": stage, "combine": stage}],
        "ffn_balanced": [{"shape": "C1", "E_loc": 8, "d": 64, "f": 64, "tokens_per_expert": 512, "us_per_expert": 1.0,
                          "TFLOP/s": 1.0, "frac_sustained": 0.1, "frac_burst": 0.1, "frac_of_per_expert_roofline": 0.1}],
        "ffn_mixed": [{"shape": "C3", "rows_per_expert": "1 x 32", "rows": 32, "active_experts": 1, "us": 39.0,
                       "weight_TB/s": 2.26, "TFLOP/s": 72.3}],
        "fused_scatter": [{"config": "C1", "ffn_plus_combine_us": 1.0, "fused_scatter_us": 1.0, "speedup": 1.0}],
        "layer": [{"config": "C1", "eager_us": 1.0, "graph_us": 1.0, "tokens_per_s_eager": 1, "tokens_per_s_graph": 1}],
        "profile": {"C2": {"E_loc": 2, "d": 64, "f": 64, "rows": [
            {"mode": 0, "tokens_per_expert": 1, "latency_us": 1.0, "p10_us": 0.9, "p90_us": 1.1, "weight_stream_floor_us": 0.5},
            {"mode": 1, "tokens_per_expert": 1, "latency_us": 2.0, "p10_us": 1.9, "p90_us": 2.1, "weight_stream_floor_us": None}]}},
        "rack_projection": [{"G": 8, "experts_per_gpu": 32, "gain_latency_vs_token_median": 0.1,
                             "gain_latency_vs_token_min": 0.0, "gain_latency_vs_token_max": 0.2,
                             "gain_latency_vs_contiguous_median": 0.5, "latency_balanced_max_over_mean_median": 1.0}],
    })
    report.write_markdown(rep, str(p), "cmd")
    text = p.read_text()
    for needle in ("## stages", "## ffn_balanced", "## ffn_mixed", "## fused_scatter", "## layer", "## profile", "## rack_projection"):
        assert needle in text
    assert os.path.getsize(p) > 500


def test_rack_projection_sweep_against_the_oracle():
    """P:L337-L347 (Fig. 15): the rack-scale projection is an evaluator sweep over G.  report.rack_sweep (C-ABI
    placement calls) against the same sweep written with the oracle's placement functions, G = 8, 32, 128."""
    import numpy as np
    from oracle import vibe_oracle as O
    from paper_2606_00735_b200 import binding as B
    from paper_2606_00735_b200 import inputs as I
    E, k, T = 256, 8, 512
    kw = dict(num_experts=E, top_k=k)
    load = O.route_topk(I.make_logits(T, E, 1.2, 7, 1.0), **kw)[2].astype(np.float64)
    tokens = [1.0, 8.0, 64.0, 512.0, 4096.0]
    lat = [13.0, 13.2, 14.5, 40.0, 300.0]                       # a weight-streaming floor, then linear growth
    Gs, seeds = (8, 32, 128), range(3)
    got = report.rack_sweep(load, B.LatencyModel(tokens, lat, 32), E, Gs, seeds)
    om = O.LatencyModel(tokens, lat, 32)
    for row, G in zip(got, Gs):
        gt, gc, ratio = [], [], []
        for seed in seeds:
            scale = I.make_throughput_scales(G, 100 + seed)
            cap = E // G
            tb = O.placement_token_balanced(load, G, cap)
            lb = O.placement_greedy(load, G, scale, om, cap)
            ct = O.placement_contiguous(E, G)
            s_tb = O.placement_eval(tb, load, G, scale, om, O.MODEL_B)[0]
            s_lb, per = O.placement_eval(lb, load, G, scale, om, O.MODEL_B)
            s_ct = O.placement_eval(ct, load, G, scale, om, O.MODEL_B)[0]
            gt.append(1.0 - s_lb / s_tb); gc.append(1.0 - s_lb / s_ct); ratio.append(s_lb / float(np.mean(per)))
        assert row["G"] == G and row["experts_per_gpu"] == E // G
        assert row["gain_latency_vs_token_median"] == round(float(np.median(gt)), 4)
        assert row["gain_latency_vs_token_min"] == round(float(min(gt)), 4)
        assert row["gain_latency_vs_token_max"] == round(float(max(gt)), 4)
        assert row["gain_latency_vs_contiguous_median"] == round(float(np.median(gc)), 4)
        assert row["latency_balanced_max_over_mean_median"] == round(float(np.median(ratio)), 4)
    # the paper's qualitative claim: with fewer experts per GPU the straggler dominates whatever the policy
    assert got[-1]["latency_balanced_max_over_mean_median"] > got[0]["latency_balanced_max_over_mean_median"]
