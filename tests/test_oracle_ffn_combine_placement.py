"""Pins for the oracle's FFN / combine / latency model / placement (O3-O8) -- CPU only."""
import itertools
import json
import os

import numpy as np
import pytest
import torch

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import inputs as I


# ---------------------------------------------------------------- bf16 helpers
def test_bf16_rounding_against_torch():
    x = I._rng(0, 9).standard_normal(200000) * np.exp(I._rng(0, 10).uniform(-20, 20, 200000))
    # torch rounds f64 -> bf16 via f32 (double rounding), so pin on f32-representable inputs,
    # where torch's f32 -> bf16 conversion is a single round-to-nearest-even
    x32 = x.astype(np.float32)
    got = O.f64_to_bf16_bits(x32.astype(np.float64))
    want = torch.from_numpy(x32).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(got, want)
    # and the oracle rounds ONCE from f64: a value a hair below a bf16 tie goes down even
    # though rounding through f32 first would land on the tie and go to even (up)
    below_tie = float.fromhex("-0x1.c2ffff3415e61p-29")      # tie would be -0x1.c3p-29
    assert O.bf16_round_f64(np.array([below_tie]))[0] == float.fromhex("-0x1.c2p-29")
    above_tie = float.fromhex("-0x1.0500002058110p-23")      # tie is -0x1.05p-23 -> even is 1.04
    assert O.bf16_round_f64(np.array([above_tie]))[0] == float.fromhex("-0x1.06p-23")
    # ties to even, exactly representable values, zero
    t = np.array([1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0, 0.0, -1.0 - 2.0 ** -8])
    assert O.bf16_round_f64(t).tolist() == [1.0, 1.0 + 2.0 ** -6, 1.0, 0.0, -1.0]
    b = np.arange(0, 0x7F80, 7, dtype=np.uint16)       # all finite positive patterns (stride 7)
    assert np.array_equal(O.f64_to_bf16_bits(O.bf16_bits_to_f64(b)), b)


# ---------------------------------------------------------------- a4 FFN
def test_ffn_matches_naive_triple_loop_tiny():
    d, f, n = 16, 24, 5
    x = I.make_X(n, d, 1)
    W1 = I.make_expert_weight(1, 0, d, f, d ** -0.5, 1)
    W3 = I.make_expert_weight(3, 0, d, f, d ** -0.5, 1)
    W2 = I.make_expert_weight(2, 0, f, d, f ** -0.5, 1)
    y, h = O.swiglu_ffn_rows(x, W1, W3, W2)
    yn = O.ffn_naive_triple_loop(x, W1, W3, W2)
    assert np.max(np.abs(y - yn)) < 1e-12


def test_ffn_single_expert_is_dense_swiglu_mlp_torch_fp64():
    """E=1 reduces to a dense SwiGLU MLP: two library matmuls + torch's silu (fp64)."""
    cfg = I.scaled(I.C0, E=1, E_loc=1, k=1, T=40)
    W1, W3, W2 = I.make_weights(1, cfg.d, cfg.f, 2)
    X = I.make_X(cfg.T, cfg.d, 2)
    ids = np.zeros((cfg.T, 1), np.int32)
    off, r2a, a2r, Xp, R = O.permute(X, ids, None, 1, 1)
    Y, H = O.grouped_ffn(Xp, off, r2a, W1, W3, W2, round_h=False)
    tx = torch.from_numpy(O.bf16_bits_to_f64(X))
    t1, t3, t2 = (torch.from_numpy(O.bf16_bits_to_f64(w[0])) for w in (W1, W3, W2))
    want = (torch.nn.functional.silu(tx @ t1) * (tx @ t3)) @ t2
    assert np.max(np.abs(Y - want.numpy())) < 1e-12
    # with the operand rounding of H the result moves by at most ~2^-9 relative per term
    Yr, _ = O.grouped_ffn(Xp, off, r2a, W1, W3, W2, round_h=True)
    m = O.ffn_error_metrics(Yr, want.numpy())
    assert 0 < m["max_abs_err_over_rms"] < 2e-2 and m["mean_rel_err"] < 5e-3


def test_ffn_up_constant_one_gives_silu_of_gate():
    d, f, n = 32, 16, 7
    x = I.make_X(n, d, 3)
    W1 = I.make_expert_weight(1, 0, d, f, d ** -0.5, 3)
    # W3 such that u == 1 for every row is impossible for random x; instead make x's first
    # column 1 and W3 = e_0 1^T : u = x[:,0] = 1
    xf = I.bf16_bits_to_f32(x).copy()
    xf[:, 0] = 1.0
    x = I.f32_to_bf16_bits(xf)
    W3f = np.zeros((d, f), np.float32)
    W3f[0, :] = 1.0
    W3 = I.f32_to_bf16_bits(W3f)
    W2 = I.f32_to_bf16_bits(np.eye(f, d, dtype=np.float32))
    y, h = O.swiglu_ffn_rows(x, W1, W3, W2, round_h=False)
    g = O.bf16_bits_to_f64(x) @ O.bf16_bits_to_f64(W1)
    silu = torch.nn.functional.silu(torch.from_numpy(g)).numpy()
    assert np.max(np.abs(h - silu)) < 1e-14
    assert np.max(np.abs(y[:, :f] - silu)) < 1e-14 and np.all(y[:, f:] == 0)


def test_ffn_empty_experts_padding_and_equivariance():
    cfg = I.scaled(I.C0, T=48)
    L = I.make_layer(cfg, 4)
    ids, w, cnt = O.route_topk(L["logits"], cfg.E, cfg.k)
    emap = np.arange(cfg.E, dtype=np.int32)
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, emap, cfg.E, 16)
    Y, H = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    assert np.all(Y[r2a < 0] == 0)
    # permutation equivariance: shuffling tokens permutes the combined outputs
    out = O.combine(Y, a2r, w, cfg.T, cfg.k)
    perm = I._rng(4, 77).permutation(cfg.T)
    ids_p, w_p, _ = O.route_topk(L["logits"][perm], cfg.E, cfg.k)
    off2, r2a2, a2r2, Xp2, _ = O.permute(L["X"][perm], ids_p, emap, cfg.E, 1)
    Y2, _ = O.grouped_ffn(Xp2, off2, r2a2, L["W1"], L["W3"], L["W2"])
    out2 = O.combine(Y2, a2r2, w_p, cfg.T, cfg.k)
    assert np.max(np.abs(out2 - out[perm])) < 1e-12


def test_grouped_ffn_row_subset_matches_full():
    cfg = I.scaled(I.C0, T=32)
    L = I.make_layer(cfg, 5)
    ids, w, _ = O.route_topk(L["logits"], cfg.E, cfg.k)
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, None, cfg.E, 1)
    Y, _ = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    rows = [0, 3, R - 1, R // 2]
    Ys, _ = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"], rows=rows)
    assert np.array_equal(Ys[rows], Y[rows])
    others = np.setdiff1d(np.arange(R), rows)
    assert np.all(np.isnan(Ys[others]))


# ---------------------------------------------------------------- a5 combine + whole layer
def test_combine_k1_unit_weight_is_unpermute():
    T, d = 9, 8
    Y = I._rng(6, 1).standard_normal((T, d))
    perm = I._rng(6, 2).permutation(T).astype(np.int32)      # assign i -> row perm[i]
    out = O.combine(Y, perm, np.ones((T, 1), np.float32), T, 1)
    assert np.array_equal(out, Y[perm])


def test_combine_linearity_and_nonresident_zero():
    T, k, d = 6, 3, 4
    Y = I._rng(7, 1).standard_normal((T * k, d))
    a2r = I._rng(7, 2).permutation(T * k).astype(np.int32)
    a2r[0:3] = -1                                            # token 0 has no resident expert
    w1 = I._rng(7, 3).uniform(0, 1, (T, k)).astype(np.float32)
    w2 = I._rng(7, 4).uniform(0, 1, (T, k)).astype(np.float32)
    o1, o2 = O.combine(Y, a2r, w1, T, k), O.combine(Y, a2r, w2, T, k)
    o12 = O.combine(Y, a2r, (w1.astype(np.float64) + w2).astype(np.float32), T, k)
    assert np.allclose(o12, o1 + o2, rtol=1e-6, atol=1e-7)
    assert np.all(o1[0] == 0)


@pytest.mark.parametrize("name", ["C0", "C3small"])
def test_full_pipeline_equals_direct_definition(name):
    """route -> permute -> grouped_ffn -> combine  ==  out[t] = sum_j w_j FFN_{id_j}(x_t)."""
    if name == "C0":
        cfg, policy = I.C0, "contiguous"
    else:
        cfg, policy = I.scaled(I.C3, T=96, d=64, f=128, E=64, E_loc=8), "random"
    L = I.make_layer(cfg, 8, map_policy=policy)
    ids, w, _ = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, L["expert_map"], cfg.E_loc, 1)
    Y, _ = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    out = O.combine(Y, a2r, w, cfg.T, cfg.k)
    direct = O.moe_layer_direct(L["X"], ids, w, L["expert_map"], L["W1"], L["W3"], L["W2"])
    assert np.max(np.abs(out - direct)) < 1e-12
    assert R > 0


# ---------------------------------------------------------------- O5 latency model
def test_latency_model_closed_forms():
    m = O.LatencyModel([1, 2, 4, 8], [10.0, 10.0, 9.0, 20.0], E_prof=4)
    assert m.per_expert(0) == 0.0
    assert m.per_expert(0.5) == 5.0                       # through the origin
    assert m.per_expert(1) == 10.0 and m.per_expert(2) == 10.0
    assert m.per_expert(4) == 10.0                        # running max repairs the dip
    assert m.per_expert(6) == 15.0
    assert m.per_expert(8) == 20.0
    assert m.per_expert(12) == 30.0                       # last slope (20-10)/(8-4) = 2.5/token
    assert m.whole_kernel(24) == 4 * m.per_expert(6)
    lin = O.LatencyModel([1.0], [1.0])
    for n in (0.0, 0.25, 1.0, 7.5, 1e6):
        assert lin.per_expert(n) == n and lin.whole_kernel(n) == n


# ---------------------------------------------------------------- O6-O8 placement
def test_placement_worked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "placement_worked_example.json")))
    lin = O.LatencyModel([1.0], [1.0])
    load, scale = g["load"], g["scale"]
    a = O.placement_greedy(load, 2, scale, lin)
    assert a.tolist() == g["greedy_assign"]
    for kind in (O.MODEL_A, O.MODEL_B):                   # linear f: A and B coincide
        sc, per = O.placement_eval(a, load, 2, scale, lin, kind)
        assert sc == pytest.approx(g["greedy_score"], rel=1e-12)
    tb = O.placement_token_balanced(load, 2)
    assert tb.tolist() == g["token_balanced_assign"]
    assert O.placement_eval(tb, load, 2, scale, lin)[0] == pytest.approx(g["token_balanced_score"], rel=1e-12)
    for cap in (0, 4):
        best, _ = O.placement_brute_force(load, 2, scale, lin, cap=cap)
        assert best == pytest.approx(g["optimum_score"], rel=1e-12)


def _direct_score(assign, load, scale, lat_fn, kind, E_prof):
    """Second, separately written evaluator straight from P:L182-L184."""
    G = len(scale)
    worst = 0.0
    for g in range(G):
        if kind == O.MODEL_A:
            n_g = sum(load[e] for e in range(len(load)) if assign[e] == g)
            t = E_prof * lat_fn(n_g / E_prof)
        else:
            t = sum(lat_fn(load[e]) for e in range(len(load)) if assign[e] == g)
        worst = max(worst, t / scale[g])
    return worst


@pytest.mark.parametrize("G,E", [(2, 8), (3, 7), (4, 6)])
def test_evaluator_matches_direct_definition_on_every_binning_and_greedy_bound(G, E):
    rng = I._rng(20 + G, E)
    load = rng.integers(0, 400, E).astype(np.float64)
    scale = I.make_throughput_scales(G, 5)
    pts_t = np.array([1, 8, 64, 256, 1024], np.float64)
    pts_l = np.array([12.0, 12.5, 14.0, 30.0, 110.0])
    model = O.LatencyModel(pts_t, pts_l, E_prof=4)
    lat = lambda n: float(np.interp(n, np.concatenate([[0], pts_t]), np.concatenate([[0], pts_l]))) if n <= 1024 \
        else 110.0 + (110.0 - 30.0) / (1024 - 256) * (n - 1024)
    for kind in (O.MODEL_A, O.MODEL_B):
        best = np.inf
        for a in itertools.product(range(G), repeat=E):
            sc, _ = O.placement_eval(a, load, G, scale, model, kind)
            assert sc == pytest.approx(_direct_score(a, load, scale, lat, kind, 4), rel=1e-12)
            best = min(best, sc)
        bf, bf_assign = O.placement_brute_force(load, G, scale, model, kind)
        assert bf == pytest.approx(best, rel=1e-12)
        greedy = O.placement_greedy(load, G, scale, model)
        assert O.placement_eval(greedy, load, G, scale, model, kind)[0] >= bf * (1 - 1e-12)


def test_greedy_special_cases():
    E, G = 64, 8
    load = np.bincount(O.route_topk(I.make_logits(2048, E, 1.2, 1), E, 8)[0].ravel(), minlength=E).astype(np.float64)
    m1 = O.LatencyModel([1, 100, 1000], [5.0, 9.0, 80.0], E_prof=8)
    m2 = O.LatencyModel([1, 50], [1.0, 2.0], E_prof=3)
    ones = np.ones(G)
    # sigma == 1  =>  identical to token-balanced
    assert np.array_equal(O.placement_greedy(load, G, ones, m1), O.placement_token_balanced(load, G))
    # tau independent of the latency model / n_ref under f_g = f/sigma_g  (M5, M6)
    sc = I.make_throughput_scales(G, 2)
    assert np.array_equal(O.placement_greedy(load, G, sc, m1), O.placement_greedy(load, G, sc, m2))
    # cap: exactly E/G per bin
    a = O.placement_greedy(load, G, sc, m1, cap=E // G)
    assert np.bincount(a, minlength=G).tolist() == [E // G] * G
    # contiguous
    assert O.placement_contiguous(8, 2).tolist() == [0, 0, 0, 0, 1, 1, 1, 1]
    # faster bins get more load
    a = O.placement_greedy(load, G, sc, m1)
    n = np.array([load[a == g].sum() for g in range(G)])
    assert np.corrcoef(n, sc)[0, 1] > 0.9
