"""GPU parity at the sizes bench.py / report.py TIME (BASELINE.json configs at full size), on sampled tokens the
oracle computes one by one: the fused scatter path, the FP8 layers (per-tensor and block-scaled), and C3's four
per-layer seeds.  Integer outputs are compared in full."""
import numpy as np
import pytest
import torch

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import binding as B
from paper_2606_00735_b200 import inputs as I

pytestmark = pytest.mark.gpu

FFN_MEAN = 5e-3
BF16_U = 2.0 ** -8


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    B.load()
    torch.cuda.set_device(0)


def dev_bf16(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def host_bits(t):
    return t.detach().view(torch.int16).cpu().numpy().view(np.uint16)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_layer_output(got, ref, ref_abs):
    """the layer bound of DESIGN.md section 4 at 1x: stated mean bar; element-wise 1e-2 RMS + the two bf16 storage terms"""
    m = O.ffn_error_metrics(got, ref)
    assert m["mean_rel_err"] <= FFN_MEAN, m
    bound = 1e-2 * m["rms_ref"] + BF16_U * ref_abs + BF16_U * np.abs(ref)
    worst = np.max(np.abs(got - ref) / bound)
    assert worst <= 1.0, (worst, m)
    return m


def device_layer(cfg, L):
    bias = dev(L["select_bias"]) if L["select_bias"] is not None else None
    rc = B.RouteConfig(select_bias=bias, **I.route_kwargs(cfg))
    emap = dev(L["expert_map"]) if cfg.E_loc < cfg.E else None
    return rc, dev(L["logits"]), dev_bf16(L["X"]), emap


def pick_sample(cfg, L, ids, n, seed, max_experts=None):
    """sampled resident tokens (first and last resident token included); with max_experts, only tokens whose
    resident experts all lie in a small set (bounds the number of experts the oracle has to quantise)"""
    em = L["expert_map"] if cfg.E_loc < cfg.E else None
    slot = ids if em is None else em[ids]
    res = np.nonzero((slot >= 0).any(axis=1))[0]
    rng = I._rng(99, seed)
    if max_experts is None:
        return sorted(set(rng.choice(res, size=min(n, len(res)), replace=False).tolist() + [int(res[0]), int(res[-1])])), slot
    cnt = np.bincount(slot[slot >= 0], minlength=cfg.E_loc)
    allowed = set(np.argsort(-cnt, kind="stable")[:max_experts].tolist())
    ok = [int(t) for t in res if all((s < 0 or int(s) in allowed) for s in slot[t])]
    assert len(ok) >= 2, "no token routed inside the allowed expert set"
    pick = rng.choice(len(ok), size=min(n, len(ok)), replace=False)
    return sorted(set([ok[i] for i in pick] + [ok[0], ok[-1]])), slot


def compact_problem(cfg, L, ids, slot, sample):
    """the mini problem the oracle solves: sampled tokens, touched experts renumbered 0..m-1"""
    touched = sorted({int(s) for t in sample for s in slot[t] if s >= 0})
    cm = {s: i for i, s in enumerate(touched)}
    em = L["expert_map"] if cfg.E_loc < cfg.E else np.arange(cfg.E, dtype=np.int32)
    emap_c = np.array([cm.get(int(em[e]), -1) if em[e] >= 0 else -1 for e in range(cfg.E)], dtype=np.int32)
    W = [np.ascontiguousarray(L[n][touched]) for n in ("W1", "W3", "W2")]
    return touched, emap_c, W, L["X"][sample], ids[sample]


# ------------------------------------------------------------------ C3: the four per-layer seeds (BJ:configs[3])
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_full_size_c3_per_layer_seeds(seed):
    """C3 draws a fresh Zipf permutation per layer (seed + layer): layers 1..3 at full size (layer 0 is
    test_full_size_layer_sampled_against_oracle[C3])."""
    cfg = I.CONFIGS["C3"]
    L = I.make_layer(cfg, seed)
    rc, lg, X, emap = device_layer(cfg, L)
    W1, W3, W2 = dev_bf16(L["W1"]), dev_bf16(L["W3"]), dev_bf16(L["W2"])
    ids_d = torch.empty((cfg.T, cfg.k), dtype=torch.int32, device="cuda")
    w_d = torch.empty((cfg.T, cfg.k), dtype=torch.float32, device="cuda")
    out, counts = B.moe_layer_forward(rc, lg, X, emap, W1, W3, W2, topk_ids=ids_d, topk_w=w_d)
    torch.cuda.synchronize()
    ids, w, c = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    assert np.array_equal(ids_d.cpu().numpy(), ids) and np.array_equal(counts.cpu().numpy(), c)
    assert np.max(np.abs(w_d.cpu().numpy().astype(np.float64) - w) / w) <= 1e-6
    sample, slot = pick_sample(cfg, L, ids, 6, seed)
    ref, ref_abs = O.moe_layer_direct(L["X"], ids, w, L["expert_map"], L["W1"], L["W3"], L["W2"], tokens=sample, return_abs=True)
    got = O.bf16_bits_to_f64(host_bits(out[sample]))
    check_layer_output(got, np.stack([ref[t] for t in sample]), np.stack([ref_abs[t] for t in sample]))


# ------------------------------------------------------------------ fused scatter path at the sizes report.py times
@pytest.mark.parametrize("name", ["C1", "C2"])
def test_full_size_scatter_path_sampled(name):
    cfg = I.CONFIGS[name]
    L = I.make_layer(cfg, 0)
    rc, lg, X, emap = device_layer(cfg, L)
    W1, W3, W2 = dev_bf16(L["W1"]), dev_bf16(L["W3"]), dev_bf16(L["W2"])
    ids_d, w_d, counts = B.route_topk(lg, rc)
    Xp, off, r2a, a2r = B.permute(X, ids_d, counts, emap, cfg.E, cfg.E_loc, 1)
    Yw = torch.full((cfg.T * cfg.k, cfg.d), float("nan"), dtype=torch.bfloat16, device="cuda")
    B.grouped_ffn_scatter(Xp, off, W1, W3, W2, r2a, w_d, Yw=Yw)
    out = B.combine_scattered(Yw, a2r, cfg.T, cfg.k)
    torch.cuda.synchronize()
    ids, w, c = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    assert np.array_equal(ids_d.cpu().numpy(), ids)
    off_o, r2a_o, a2r_o, _, _ = O.permute(np.zeros((cfg.T, 1), np.uint16), ids, None, cfg.E_loc, 1)
    assert np.array_equal(off.cpu().numpy(), off_o) and np.array_equal(a2r.cpu().numpy(), a2r_o)
    sample, slot = pick_sample(cfg, L, ids, 10, 5)
    ref, ref_abs = O.moe_layer_direct(L["X"], ids, w, None, L["W1"], L["W3"], L["W2"], tokens=sample, return_abs=True)
    got = O.bf16_bits_to_f64(host_bits(out[sample]))
    check_layer_output(got, np.stack([ref[t] for t in sample]), np.stack([ref_abs[t] for t in sample]))
    # the scattered rows themselves: Yw[t*k + j] = bf16(w_j * y_j) for two sampled tokens
    for t in sample[:2]:
        for j in range(cfg.k):
            y, _ = O.swiglu_ffn_rows(L["X"][t:t + 1], L["W1"][ids[t, j]], L["W3"][ids[t, j]], L["W2"][ids[t, j]])
            want = float(np.float32(w[t, j])) * y[0]
            g = O.bf16_bits_to_f64(host_bits(Yw[t * cfg.k + j]))
            rms = float(np.sqrt(np.mean(want * want)))
            assert np.all(np.abs(g - want) <= 1e-2 * rms + BF16_U * np.abs(want))


def per_expert(fn, W):
    """apply an oracle weight packer expert by expert (bounds the f64 temporaries at full size)"""
    parts = [fn(W[e:e + 1]) for e in range(W.shape[0])]
    return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])


# ------------------------------------------------------------------ FP8 layers at full size
def mx_reference(cfg, L, ids, w, slot, sample):
    touched, emap_c, (W1, W3, W2), Xs, ids_s = compact_problem(cfg, L, ids, slot, sample)
    Xq_tok, Xs_tok = O.mx_quantize_rows(Xs)
    off, r2a, a2r, Xpq16, _ = O.permute(Xq_tok.view(np.uint16), ids_s, emap_c, len(touched), 1)
    Xpq = np.ascontiguousarray(Xpq16).view(np.uint8)
    Xsf = Xs_tok[r2a // cfg.k]
    W1q, W1s = per_expert(O.mx_pack_weights, W1); W3q, W3s = per_expert(O.mx_pack_weights, W3); W2q, W2s = per_expert(O.mx_pack_weights, W2)
    Y, _, _ = O.grouped_ffn_mxfp8(Xpq, Xsf, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s)
    w_s = w[sample]
    return O.combine(Y, a2r, w_s, len(sample), cfg.k), O.combine(np.abs(Y), a2r, w_s, len(sample), cfg.k)


@pytest.mark.parametrize("name", ["C1", "C3"])
def test_full_size_mxfp8_layer_sampled(name):
    """vibe_moe_layer_forward_mxfp8 at full size against the oracle's block-scaled composition on sampled tokens."""
    cfg = I.CONFIGS[name]
    L = I.make_layer(cfg, 0)
    rc, lg, X, emap = device_layer(cfg, L)
    packed = []
    for n, role in (("W1", B.MX_ROLE_GATE), ("W3", B.MX_ROLE_UP), ("W2", B.MX_ROLE_DOWN)):
        Wd = dev_bf16(L[n])
        q, sf = B.mxfp8_pack_weights(Wd, role, sf=packed[0][1] if role == B.MX_ROLE_UP else None)
        packed.append((q, sf))
        del Wd
    out, counts = B.moe_layer_forward_mxfp8(rc, lg, X, emap, packed[0][0], packed[1][0], packed[1][1], packed[2][0], packed[2][1])
    torch.cuda.synchronize()
    ids, w, c = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    assert np.array_equal(counts.cpu().numpy(), c)
    sample, slot = pick_sample(cfg, L, ids, 8, 11, max_experts=2 if name == "C1" else 6)
    ref, ref_abs = mx_reference(cfg, L, ids, w, slot, sample)
    check_layer_output(O.bf16_bits_to_f64(host_bits(out[sample])), ref, ref_abs)


@pytest.mark.parametrize("name", ["C1", "C3"])
def test_full_size_fp8_layer_sampled(name):
    """vibe_moe_layer_forward_fp8 (per-expert / per-row scales) at full size.  h_scale is CALIBRATED: 4 x the oracle's
    max |H| of the bf16 FFN over the sampled rows of each touched expert, / 448 (untouched experts get the mean) --
    the sampled rows then cannot saturate, and their outputs do not depend on the other experts' scales."""
    cfg = I.CONFIGS[name]
    L = I.make_layer(cfg, 0)
    rc, lg, X, emap = device_layer(cfg, L)
    ids, w, c = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    sample, slot = pick_sample(cfg, L, ids, 8, 12, max_experts=2 if name == "C1" else 6)
    touched, emap_c, (W1, W3, W2), Xs, ids_s = compact_problem(cfg, L, ids, slot, sample)
    off_b, r2a_b, _, Xp_b, _ = O.permute(Xs, ids_s, emap_c, len(touched), 1)
    _, H_bf = O.grouped_ffn(Xp_b, off_b, r2a_b, W1, W3, W2)
    hs_c = np.array([4.0 * np.abs(H_bf[off_b[i]:off_b[i + 1]]).max() / 448.0 for i in range(len(touched))], np.float32)
    hs = np.full(cfg.E_loc, float(hs_c.mean()), np.float32)
    hs[touched] = hs_c
    packs = [B.fp8_pack_weights(dev_bf16(L[n])) for n in ("W1", "W3", "W2")]
    out, counts = B.moe_layer_forward_fp8(rc, lg, X, emap, packs[0][0], packs[0][1], packs[1][0], packs[1][1], packs[2][0],
                                          packs[2][1], dev(hs))
    torch.cuda.synchronize()
    assert np.array_equal(counts.cpu().numpy(), c)
    Xq_tok, ts = O.fp8_quantize_rows(Xs)
    off, r2a, a2r, Xpq16, _ = O.permute(Xq_tok.view(np.uint16), ids_s, emap_c, len(touched), 1)
    Xpq = np.ascontiguousarray(Xpq16).view(np.uint8)
    rs = ts[r2a // cfg.k]
    W1q, s1 = per_expert(O.fp8_pack_weights, W1); W3q, s3 = per_expert(O.fp8_pack_weights, W3); W2q, s2 = per_expert(O.fp8_pack_weights, W2)
    for i, e in enumerate(touched):                       # the packed scales of the GPU are those of the oracle
        assert packs[0][1][e].item() == s1[i] and packs[2][1][e].item() == s2[i]
    Y, _ = O.grouped_ffn_fp8(Xpq, rs, off, r2a, W1q, s1, W3q, s3, W2q, s2, hs_c)
    w_s = w[sample]
    ref, ref_abs = O.combine(Y, a2r, w_s, len(sample), cfg.k), O.combine(np.abs(Y), a2r, w_s, len(sample), cfg.k)
    check_layer_output(O.bf16_bits_to_f64(host_bits(out[sample])), ref, ref_abs)
