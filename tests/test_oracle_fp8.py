"""Pins for the oracle's FP8 (e4m3) quantisers and FP8 grouped FFN (O11; f2) -- CPU only."""
import numpy as np
import pytest
import torch

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import inputs as I


def test_e4m3_table_against_torch_and_closed_forms():
    t = O.e4m3_decode_table()
    want = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(np.isnan(t), np.isnan(want)) and np.isnan(t).sum() == 2
    ok = ~np.isnan(t)
    assert np.array_equal(t[ok], want[ok])
    assert t[0x7E] == 448.0 and t[0x01] == 2.0 ** -9 and t[0x08] == 2.0 ** -6 and t[0x38] == 1.0 and t[0xB8] == -1.0
    assert np.all(np.diff(t[0:0x7F]) > 0)                      # positive codes are ordered


def test_e4m3_encode_against_torch_roundtrip_ties_and_saturation():
    t = O.e4m3_decode_table()
    codes = np.array([c for c in range(256) if (c & 0x7F) != 0x7F], dtype=np.uint8)
    assert np.array_equal(O.e4m3_encode(t[codes]) & 0x7F, codes & 0x7F)                    # exact values round-trip
    assert np.array_equal(O.e4m3_encode(t[codes])[t[codes] != 0], codes[t[codes] != 0])    # with their sign
    rng = I._rng(8, 8)
    x = np.concatenate([rng.standard_normal(20000) * np.exp(rng.uniform(-12, 7, 20000)),
                        [0.0, 448.0, 449.0, 1e9, -1e9, 2.0 ** -10, 3 * 2.0 ** -10, 2.0 ** -9 * 7.5, 464.0, 480.0]])
    x32 = x.astype(np.float32)                                  # torch converts from f32: pin on f32-representable inputs
    got = O.e4m3_encode(x32.astype(np.float64))
    sat = np.clip(x32, -448.0, 448.0)                           # torch's cast does not saturate (448 < |x| -> NaN): clamp first
    want = torch.from_numpy(sat).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(got, want)
    # ties to even: 17 = midway between 16 (m=0) and 18 (m=1) -> 16; 19 midway 18/20 -> 20; subnormal tie 2^-10 -> 0
    assert t[O.e4m3_encode(np.array([17.0, 19.0, 2.0 ** -10, 3 * 2.0 ** -10]))].tolist() == [16.0, 20.0, 0.0, 2.0 ** -8]
    # brute force nearest-value search on random inputs
    pos = t[:0x7F]
    for v in np.abs(x[:300]):
        v = min(v, 448.0)
        c = int(O.e4m3_encode(np.array([v]))[0])
        assert abs(pos[c] - v) == np.min(np.abs(pos - v))


def test_fp8_quantisers_scales_and_layout():
    d, f, E, R = 64, 48, 3, 10
    W = np.stack([I.make_expert_weight(1, e, d, f, 0.3 * (e + 1), 2) for e in range(E)])
    W[2] = 0                                                    # an all-zero expert keeps scale 1
    codes, scale = O.fp8_pack_weights(W)
    assert codes.shape == (E, f, d) and scale.dtype == np.float32 and scale[2] == 1.0 and np.all(codes[2] & 0x7F == 0)
    Wf = O.bf16_bits_to_f64(W)
    t = O.e4m3_decode_table()
    for e in range(2):
        assert scale[e] == np.float32(np.abs(Wf[e]).max() / 448.0)
        deq = t[codes[e]].T * np.float64(scale[e])
        assert np.max(np.abs(deq)) <= np.abs(Wf[e]).max() * (1 + 1e-6)
        assert np.all(np.abs(deq - Wf[e]) <= 2.0 ** -4 * np.abs(Wf[e]) + 2.0 ** -10 * np.float64(scale[e]))   # half an ulp (3 mantissa bits)
        assert np.abs(t[codes[e]]).max() == 448.0               # the largest element maps to the largest code
    X = I.make_X(R, d, 3)
    X[4] = 0
    xq, rs = O.fp8_quantize_rows(X)
    Xf = O.bf16_bits_to_f64(X)
    assert rs[4] == 1.0 and np.all(xq[4] & 0x7F == 0)
    for r in (0, 9):
        assert rs[r] == np.float32(np.abs(Xf[r]).max() / 448.0) and np.abs(t[xq[r]]).max() == 448.0


def test_fp8_ffn_reduces_to_the_plain_definition():
    """On inputs that ARE e4m3 values with unit scales, the FP8 FFN is the plain SwiGLU FFN followed by one
    e4m3 rounding of H: checked against an independent torch fp64 computation; and the scales factor out."""
    rng = I._rng(9, 9)
    t = O.e4m3_decode_table()
    E, n, d, f = 2, 7, 32, 24
    pick = lambda shape: rng.integers(0x20, 0x40, shape).astype(np.uint8) | (rng.integers(0, 2, shape).astype(np.uint8) << 7)
    Xq, W1q, W3q, W2q = pick((E * n, d)), pick((E, f, d)), pick((E, f, d)), pick((E, d, f))
    off = np.array([0, n, 2 * n]); r2a = np.arange(E * n)
    one = np.ones(E, np.float32)
    hs = np.array([0.5, 2.0], np.float32)
    Y, Hq = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), off, r2a, W1q, one, W3q, one, W2q, one, hs)
    for e in range(E):
        x = torch.from_numpy(t[Xq[e * n:(e + 1) * n]])
        g = x @ torch.from_numpy(t[W1q[e]]).T
        u = x @ torch.from_numpy(t[W3q[e]]).T
        h = (torch.nn.functional.silu(g) * u).numpy()
        hq = O.e4m3_encode(h / float(hs[e]))
        assert np.array_equal(hq, Hq[e * n:(e + 1) * n])
        y = (t[hq] @ t[W2q[e]].T) * float(hs[e])
        assert np.allclose(Y[e * n:(e + 1) * n], y, rtol=1e-12, atol=0)
    # scales factor out of the down projection: doubling s2 doubles Y; an empty expert gives zero rows
    Y2, _ = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), off, r2a, W1q, one, W3q, one, W2q, 2 * one, hs)
    assert np.allclose(Y2, 2 * Y, rtol=1e-12)
    Y3, _ = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), np.array([0, 0, 2 * n]), r2a, W1q, one, W3q, one, W2q, one, hs)
    assert Y3.shape == Y.shape


def test_fp8_pipeline_close_to_the_bf16_ffn():
    """Quantise -> FP8 FFN is an approximation of the bf16 FFN: within the error e4m3's 3 mantissa bits allow."""
    cfg = I.scaled(I.C0, T=24, d=64, f=64, E=2, E_loc=2, k=1)
    L = I.make_layer(cfg, 4)
    ids = (np.arange(cfg.T) % 2).astype(np.int32)[:, None]
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, None, 2, 1)
    Y_ref, H_ref = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    W1q, s1 = O.fp8_pack_weights(L["W1"]); W3q, s3 = O.fp8_pack_weights(L["W3"]); W2q, s2 = O.fp8_pack_weights(L["W2"])
    Xq, rs = O.fp8_quantize_rows(Xp)
    hs = np.array([np.abs(H_ref[off[e]:off[e + 1]]).max() / 448.0 for e in range(2)], np.float32)
    Y, _ = O.grouped_ffn_fp8(Xq, rs, off, r2a, W1q, s1, W3q, s3, W2q, s2, hs)
    m = O.ffn_error_metrics(Y, Y_ref)
    assert m["mean_rel_err"] < 0.08 and m["max_abs_err_over_rms"] < 0.5, m
