"""GPU parity of the BLOCK-SCALED FP8 path (S8(f) f2 as written: "e4m3, block-scaled"; readings Q5-Q8) against the
oracle's O12, through the C ABI.  Bars: codes and scale bytes of the quantisers bit-exact; H (a block-quantised
intermediate decided by an fp32 value on the GPU, by binary32(f64) in the oracle) compared after dequantisation;
Y and the layer output at the STATED north-star bars (max|err| <= 2e-2 RMS, mean rel <= 5e-3; the layer output with
the storage-rounding terms of DESIGN.md section 4)."""
import numpy as np
import pytest
import torch

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import binding as B
from paper_2606_00735_b200 import inputs as I

pytestmark = pytest.mark.gpu

FFN_MAX = 2e-2
FFN_MEAN = 5e-3
BF16_U = 2.0 ** -8
ALIGN = B.MX_ROW_ALIGN


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


def read_sf(flat, which, rows, K, R_cap=0, role=B.MX_ROLE_DOWN, E=1):
    """device scale array in layout `which` -> row-major uint8 [E, rows, K/32] (pure index gather)"""
    flat = flat.cpu().numpy()
    idx = B.mxfp8_sf_offsets(which, rows, K, R_cap, role).numpy()
    per = B.mxfp8_sf_bytes(which, rows if which != B.MX_SF_TOKENS else max(R_cap, rows), K, 1)
    return np.stack([flat[e * per + idx] for e in range(E)])


def to_tokens_layout(sf_rows, R_cap, K):
    """row-major [R, K/32] -> flat TOKENS-layout array for R_cap rows (index scatter only), rest = 127"""
    R = sf_rows.shape[0]
    flat = np.full(max(16, B.mxfp8_sf_bytes(B.MX_SF_TOKENS, R_cap, K)), 127, np.uint8)
    flat[B.mxfp8_sf_offsets(B.MX_SF_TOKENS, R, K, R_cap).numpy()] = sf_rows
    return flat


def weight_layouts(W1s, W3s, W2s, d, f, E):
    """oracle row-major weight scales [E,N,K/32] -> the flat GATE_UP and DOWN arrays the kernel reads"""
    sf13 = np.full(max(16, B.mxfp8_sf_bytes(B.MX_SF_GATE_UP, f, d, E)), 127, np.uint8)
    sf2 = np.full(max(16, B.mxfp8_sf_bytes(B.MX_SF_DOWN, d, f, E)), 127, np.uint8)
    p13, p2 = B.mxfp8_sf_bytes(B.MX_SF_GATE_UP, f, d, 1), B.mxfp8_sf_bytes(B.MX_SF_DOWN, d, f, 1)
    ig = B.mxfp8_sf_offsets(B.MX_SF_GATE_UP, f, d, role=B.MX_ROLE_GATE).numpy()
    iu = B.mxfp8_sf_offsets(B.MX_SF_GATE_UP, f, d, role=B.MX_ROLE_UP).numpy()
    idn = B.mxfp8_sf_offsets(B.MX_SF_DOWN, d, f).numpy()
    for e in range(E):
        sf13[e * p13 + ig] = W1s[e]
        sf13[e * p13 + iu] = W3s[e]
        sf2[e * p2 + idn] = W2s[e]
    return sf13, sf2


@pytest.mark.parametrize("block", [32, 128])
def test_mx_quantisers_bit_exact(block):
    rng = I._rng(31, block)
    R, d = 333, 512
    X = I.make_X(R, d, 7)
    X[17] = 0
    X[5, :] = I.f32_to_bf16_bits((rng.standard_normal(d) * 1e-3).astype(np.float32))
    X[6, :] = I.f32_to_bf16_bits((rng.standard_normal(d) * np.exp(rng.uniform(-30, 30, d))).astype(np.float32))
    xq_o, xs_o = O.mx_quantize_rows(X, block)
    xq, xs = B.mxfp8_quantize_rows(dev_bf16(X), block)
    torch.cuda.synchronize()
    assert np.array_equal(xq.cpu().numpy(), xq_o), "activation codes"
    assert np.array_equal(xs.cpu().numpy(), xs_o), "activation scale bytes (row-major)"
    xq2, xs2 = B.mxfp8_quantize_rows(dev_bf16(X), block, B.MX_SF_TOKENS, R_cap=400)
    torch.cuda.synchronize()
    assert np.array_equal(xq2.cpu().numpy(), xq_o)
    assert np.array_equal(read_sf(xs2, B.MX_SF_TOKENS, R, d, R_cap=400)[0], xs_o), "scale bytes (TOKENS layout)"
    E, K, N = 3, 256, 384
    W = np.stack([I.make_expert_weight(1, e, K, N, 0.05 * (e + 1), 8) for e in range(E)])
    W[1] = 0
    wq_o, ws_o = O.mx_pack_weights(W, block)
    Wd = dev_bf16(W)
    wq, sfd = B.mxfp8_pack_weights(Wd, B.MX_ROLE_DOWN, block)
    wg, sfg = B.mxfp8_pack_weights(Wd, B.MX_ROLE_GATE, block)
    wu, sfg = B.mxfp8_pack_weights(Wd, B.MX_ROLE_UP, block, sf=sfg)
    torch.cuda.synchronize()
    for w in (wq, wg, wu):
        assert np.array_equal(w.cpu().numpy(), wq_o), "weight codes / [E,N,K] layout"
    assert np.array_equal(read_sf(sfd, B.MX_SF_DOWN, N, K, E=E), ws_o), "weight scales (DOWN layout)"
    assert np.array_equal(read_sf(sfg, B.MX_SF_GATE_UP, N, K, role=B.MX_ROLE_GATE, E=E), ws_o), "weight scales (GATE half)"
    assert np.array_equal(read_sf(sfg, B.MX_SF_GATE_UP, N, K, role=B.MX_ROLE_UP, E=E), ws_o), "weight scales (UP half)"


def run_ffn_case(off, r2a, Xp, W1, W3, W2, extra_rows=64):
    """oracle and GPU block-scaled FFN on the same permuted rows (offsets multiples of 64)."""
    E = len(off) - 1
    R = int(off[-1])
    d, f = W1.shape[1], W1.shape[2]
    W1q, W1s = O.mx_pack_weights(W1); W3q, W3s = O.mx_pack_weights(W3); W2q, W2s = O.mx_pack_weights(W2)
    Xq, Xs = O.mx_quantize_rows(Xp)
    Y_o, Hq_o, Hs_o = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s)
    Rcap = R + extra_rows
    Xq_d = torch.full((Rcap, d), 0x7E, dtype=torch.uint8, device="cuda")     # 448s past the end must not leak
    Xq_d[:R] = dev(Xq)
    xsf = to_tokens_layout(Xs, Rcap, d)
    sf13, sf2 = weight_layouts(W1s, W3s, W2s, d, f, E)
    Y, Hq, Hsf = B.grouped_ffn_mxfp8(Xq_d, dev(xsf), dev(off), dev(W1q), dev(W3q), dev(sf13), dev(W2q), dev(sf2))
    torch.cuda.synchronize()
    real = np.nonzero(r2a[:R] >= 0)[0]
    hs = read_sf(Hsf, B.MX_SF_TOKENS, R, f, R_cap=Rcap)[0]
    H_gpu = O.mx_dequantize(Hq.cpu().numpy()[:R][real], hs[real])
    H_ref = O.mx_dequantize(Hq_o[real], Hs_o[real])
    # GEMM-2 in isolation: the device's Y against the oracle's down projection of the DEVICE's own H codes and scales
    # (no code decision in between: fp32 accumulation order + the bf16 storage of Y, element by element)
    Y_own = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s, H_given=(Hq.cpu().numpy()[:R], hs))[0][real]
    got = O.bf16_bits_to_f64(host_bits(Y)[:R][real])
    assert np.all(np.abs(got - Y_own) <= 2.0 ** -8 * np.abs(Y_own) + 1e-3 * float(np.sqrt(np.mean(Y_own ** 2))))
    return Y_o, Y, H_ref, H_gpu, hs[real], Hs_o[real], real, R


def check_ffn_outputs(Y_o, Y, H_ref, H_gpu, hs, hs_o, real, R):
    # H: identical codes except where fp32 and binary32(f64) values straddle a rounding or a block-exponent boundary.
    # Element-wise: one e4m3 step of the LARGER of the two block scales (2^-3 relative of the value + one subnormal step)
    diff_blocks = float((hs != hs_o).mean())
    assert diff_blocks <= 2e-3, f"{diff_blocks:.5f} of the H blocks chose another exponent"
    step = np.repeat(np.ldexp(1.0, np.maximum(hs, hs_o).astype(np.int64) - 127), 32, axis=-1)
    tol = 2.0 ** -3 * np.maximum(np.abs(H_ref), np.abs(H_gpu)) + 2.0 ** -9 * step
    assert np.all(np.abs(H_gpu - H_ref) <= tol * 1.0001)
    frac = float((H_gpu != H_ref).mean())
    assert frac <= 5e-3, f"{frac:.5f} of the dequantised H values differ"
    got = O.bf16_bits_to_f64(host_bits(Y)[:R][real])
    m = O.ffn_error_metrics(got, Y_o[real])
    assert m["max_abs_err_over_rms"] <= FFN_MAX and m["mean_rel_err"] <= FFN_MEAN, m
    return m


@pytest.mark.parametrize("T,E,k,d,f", [(64, 8, 2, 256, 512), (700, 4, 2, 384, 256), (300, 16, 4, 128, 128),
                                       (1500, 2, 1, 512, 640)])
def test_ffn_mxfp8_against_oracle(T, E, k, d, f):
    cfg = I.scaled(I.C0, T=T, E=E, E_loc=E, k=k, d=d, f=f)
    L = I.make_layer(cfg, 3)
    ids, w, _ = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, None, E, ALIGN)
    check_ffn_outputs(*run_ffn_case(off, r2a, Xp, L["W1"], L["W3"], L["W2"]))


@pytest.mark.parametrize("rows,d,f", [([1, 15, 16, 17, 0, 31, 33, 255], 128, 256), ([4100, 790, 0, 385, 192, 193, 449, 64, 65], 128, 512)])
def test_ffn_mxfp8_ragged_token_tiles(rows, d, f):
    """ragged segments padded to 64-row starts: 1 / 16 / 17 / 33 rows, empty experts, exact multiples of the 192-row
    tile and one more, several tiles with a tail"""
    E = len(rows)
    pad = [(n + ALIGN - 1) // ALIGN * ALIGN for n in rows]
    off = np.concatenate([[0], np.cumsum(pad)]).astype(np.int32)
    R = int(off[-1])
    r2a = np.full(R, -1, np.int32)
    for e, n in enumerate(rows):
        r2a[off[e]:off[e] + n] = np.arange(n)
    Xp = I.make_X(R, d, 79)
    Xp[r2a < 0] = 0                                                      # padding rows are zero rows (P2)
    W1, W3, W2 = I.make_weights(E, d, f, 80)
    check_ffn_outputs(*run_ffn_case(off, r2a, Xp, W1, W3, W2, extra_rows=300))


@pytest.mark.parametrize("which", ["C2s", "C3s"])
def test_layer_forward_mxfp8_against_oracle(which):
    """vibe_moe_layer_forward_mxfp8 against the oracle's composition: route -> block-32 quantisation of the token
    rows -> stable permutation (align 64) of the code rows and of their scale rows -> MX FFN -> combine.  Held to the
    layer bound of DESIGN.md section 4 at 1x (no doubling)."""
    cfg = {"C2s": I.scaled(I.C2, T=500, d=256, f=384, E=16, E_loc=16, k=4),
           "C3s": I.scaled(I.C3, T=700, d=384, f=128, E=64, E_loc=8, k=6, n_group=8, topk_group=4)}[which]
    L = I.make_layer(cfg, 9, map_policy="random" if cfg.E_loc < cfg.E else "contiguous")
    kw = I.route_kwargs(cfg)
    ids_o, w_o, c_o = O.route_topk(L["logits"], select_bias=L["select_bias"], **kw)
    em = L["expert_map"] if cfg.E_loc < cfg.E else None
    Xq_tok, Xs_tok = O.mx_quantize_rows(L["X"])
    off, r2a, a2r, Xpq16, R = O.permute(Xq_tok.view(np.uint16), ids_o, em, cfg.E_loc, ALIGN)
    Xpq = np.ascontiguousarray(Xpq16).view(np.uint8)
    Xs = np.full((int(off[-1]), cfg.d // 32), 127, np.uint8)
    real = r2a >= 0
    Xs[real] = Xs_tok[r2a[real] // cfg.k]
    W1q, W1s = O.mx_pack_weights(L["W1"]); W3q, W3s = O.mx_pack_weights(L["W3"]); W2q, W2s = O.mx_pack_weights(L["W2"])
    Y_o, _, _ = O.grouped_ffn_mxfp8(Xpq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s)
    ref = O.combine(Y_o, a2r, w_o, cfg.T, cfg.k)
    ref_abs = O.combine(np.abs(Y_o), a2r, w_o, cfg.T, cfg.k)
    bias = dev(L["select_bias"]) if L["select_bias"] is not None else None
    rc = B.RouteConfig(select_bias=bias, **kw)
    Wd = [dev_bf16(L[n]) for n in ("W1", "W3", "W2")]
    W1d, sf13 = B.mxfp8_pack_weights(Wd[0], B.MX_ROLE_GATE)
    W3d, sf13 = B.mxfp8_pack_weights(Wd[1], B.MX_ROLE_UP, sf=sf13)
    W2d, sf2 = B.mxfp8_pack_weights(Wd[2], B.MX_ROLE_DOWN)
    out, counts = B.moe_layer_forward_mxfp8(rc, dev(L["logits"]), dev_bf16(L["X"]), dev(em) if em is not None else None,
                                            W1d, W3d, sf13, W2d, sf2)
    torch.cuda.synchronize()
    assert np.array_equal(counts.cpu().numpy(), c_o)
    got = O.bf16_bits_to_f64(host_bits(out))
    m = O.ffn_error_metrics(got, ref)
    assert m["mean_rel_err"] <= FFN_MEAN, m
    bound = 1e-2 * m["rms_ref"] + BF16_U * ref_abs + BF16_U * np.abs(ref)
    assert np.all(np.abs(got - ref) <= bound), (np.max(np.abs(got - ref) / bound), m)


def test_profile_expert_latency_mxfp8_sanity():
    """a6 for the block-scaled FFN: positive, finite, a step function of n with steps of 64 rows (segments are
    padded to the scale-factor row alignment), growing with n, not faster than the nominal dense FP8 peak."""
    cfg = I.scaled(I.C2, E=16, E_loc=16)
    Wb = [dev_bf16(x) for x in I.make_weights(cfg.E_loc, cfg.d, cfg.f, 0)]
    W1m, sf13 = B.mxfp8_pack_weights(Wb[0], B.MX_ROLE_GATE)
    W3m, sf13 = B.mxfp8_pack_weights(Wb[1], B.MX_ROLE_UP, sf=sf13)
    W2m, sf2 = B.mxfp8_pack_weights(Wb[2], B.MX_ROLE_DOWN)
    sweep = [1, 64, 128, 2048]
    lat = B.profile_expert_latency_mxfp8(W1m, W3m, sf13, W2m, sf2, sweep, mode=0, warmup=3, iters=21)
    assert lat.shape == (4,) and np.all(lat > 0) and np.all(np.isfinite(lat))
    assert abs(lat[0] - lat[1]) <= 0.15 * lat[1], lat            # 1 row and 64 rows are the same launch
    assert lat[3] > lat[2] >= lat[1] * 0.9, lat
    assert lat[3] * 1e-6 >= 6.0 * 2048 * cfg.d * cfg.f / 4.5e15
    solo = B.profile_expert_latency_mxfp8(W1m, W3m, sf13, W2m, sf2, [128], mode=1, warmup=2, iters=5)
    assert solo[0] > 0
