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
    # Hq_given: the down projection on given codes.  The computed codes give the same Y bit for bit; ONE code moved to
    # another e4m3 value changes exactly its row, by (new - old) * hs * w2[:, that feature] (hand formula, not the oracle's)
    Yg, Hq2 = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), off, r2a, W1q, one, W3q, one, W2q, one, hs, Hq_given=Hq)
    assert np.array_equal(Yg, Y) and np.array_equal(Hq2, Hq)
    alt = Hq.copy()
    r, c = n + 3, 5                                              # a row of expert 1
    alt[r, c] = 0x38 if Hq[r, c] != 0x38 else 0x40               # 1.0 (or 2.0)
    Ya, Hq3 = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), off, r2a, W1q, one, W3q, one, W2q, one, hs, Hq_given=alt)
    assert np.array_equal(Hq3, Hq)                               # the returned codes are the computed ones
    delta = (float(t[alt[r, c]]) - float(t[Hq[r, c]])) * float(hs[1]) * t[W2q[1]][:, c]
    assert np.allclose(Ya[r] - Y[r], delta, rtol=1e-9, atol=1e-12)
    others = np.ones(E * n, bool); others[r] = False
    assert np.array_equal(Ya[others], Y[others])


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


# ----------------------------------------------------------------------------------------------------
# round 2: the vectorised encoder, the quotient-precision pin (Q3), block-scaled FP8 (O12, Q5-Q8)
# ----------------------------------------------------------------------------------------------------
import json
import os
from fractions import Fraction

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_e4m3_encode_array_form_equals_the_elementwise_definition():
    rng = I._rng(8, 9)
    t = O.e4m3_decode_table()
    fin = t[~np.isnan(t)]
    mid = (t[:0x7E] + t[1:0x7F]) / 2                            # every tie point of the positive range
    x = np.concatenate([rng.standard_normal(30000) * np.exp(rng.uniform(-14, 8, 30000)), fin, mid, -mid,
                        np.nextafter(mid, 0), np.nextafter(mid, 1e9), [0.0, -0.0, 448.0, 449.0, 1e30, -1e30, 2.0 ** -6]])
    assert np.array_equal(O.e4m3_encode(x), O.e4m3_encode_scalar(x))


def _frac(s):
    return Fraction(s)


def _rn_binary32(q: Fraction) -> Fraction:
    """Correctly rounded (nearest, ties to even) binary32 value of a positive rational, in exact arithmetic."""
    e = 0
    while Fraction(2) ** (e + 1) <= q:
        e += 1
    while Fraction(2) ** e > q:
        e -= 1
    ulp = Fraction(2) ** (e - 23)
    n = q / ulp
    lo = n.numerator // n.denominator
    r = n - lo
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and lo % 2):
        lo += 1
    return lo * ulp


def test_quantiser_quotient_is_binary32_golden():
    """Q3 pin: tests/golden/fp8_quotient_precision_example.json.  The expected codes are re-derived here in exact
    rational arithmetic (no numpy floats), and the row is one where an f64 quotient gives OTHER codes."""
    g = json.load(open(os.path.join(GOLD, "fp8_quotient_precision_example.json")))
    vals = [_frac(v) for v in g["row_values"]]
    amax = max(abs(v) for v in vals)
    assert amax == _frac(g["amax"])
    scale = _rn_binary32(amax / 448)
    assert scale == 8987794 * Fraction(1, 2 ** 34)
    t = O.e4m3_decode_table()
    want = [int(c, 16) for c in g["expected_codes"]]
    for v, code in zip(vals, want):
        if v == 0:
            assert code == 0
            continue
        q32 = _rn_binary32(abs(v) / scale)                     # the binary32 quotient, exactly
        cands = [(abs(Fraction(float(t[c])) - q32), c & 1, c) for c in range(0x7F)]
        best = min(cands)                                      # nearest value; on a tie the even mantissa (c & 1 == 0)
        assert best[2] == (code & 0x7F) and (code >> 7) == (1 if v < 0 else 0)
    bits = np.array([int(b, 16) for b in g["row_bf16_bits"]], dtype=np.uint16)[None, :]
    assert [Fraction(float(x)) for x in O.bf16_bits_to_f64(bits)[0]] == vals
    codes, rs = O.fp8_quantize_rows(bits)
    assert Fraction(float(rs[0])) == scale
    assert codes[0].tolist() == want
    # the same rule in the static-scale quantiser used for H, and in the weight packer (one expert, K = 6, N = 1)
    assert O.fp8_quantize_static(O.bf16_bits_to_f64(bits)[0], rs[0]).tolist() == want
    wc, ws = O.fp8_pack_weights(bits.reshape(1, 6, 1))
    assert wc[0, 0].tolist() == want and ws[0] == rs[0]
    # discriminating: the f64 quotient lands elsewhere
    other = O.e4m3_encode(O.bf16_bits_to_f64(bits)[0] / np.float64(rs[0])).tolist()
    assert other == [int(c, 16) for c in g["codes_if_the_quotient_were_f64"]] and other != want


def test_fp8_ffn_h_quotient_follows_q3_against_torch():
    """H inside grouped_ffn_fp8 is quantised as Q3 says (binary32 value, binary32 quotient): the codes equal
    torch's own float32 division + float8_e4m3fn cast on an independently computed h."""
    rng = I._rng(9, 10)
    t = O.e4m3_decode_table()
    E, n, d, f = 2, 40, 32, 96
    pick = lambda shape: rng.integers(0x20, 0x40, shape).astype(np.uint8) | (rng.integers(0, 2, shape).astype(np.uint8) << 7)
    Xq, W1q, W3q, W2q = pick((E * n, d)), pick((E, f, d)), pick((E, f, d)), pick((E, d, f))
    off = np.array([0, n, 2 * n]); r2a = np.arange(E * n)
    one = np.ones(E, np.float32)
    hs = np.array([0.0371, 0.0113], np.float32)                # not powers of two
    _, Hq = O.grouped_ffn_fp8(Xq, np.ones(E * n, np.float32), off, r2a, W1q, one, W3q, one, W2q, one, hs)
    for e in range(E):
        x = torch.from_numpy(t[Xq[e * n:(e + 1) * n]])
        h = torch.nn.functional.silu(x @ torch.from_numpy(t[W1q[e]]).T) * (x @ torch.from_numpy(t[W3q[e]]).T)
        q = (h.to(torch.float32) / torch.tensor(hs[e])).clamp(-448.0, 448.0)
        assert np.array_equal(q.to(torch.float8_e4m3fn).view(torch.uint8).numpy(), Hq[e * n:(e + 1) * n])


def test_mx_block_scale_golden():
    g = json.load(open(os.path.join(GOLD, "mx_block_scale_example.json")))
    for c in g["cases"]:
        v = np.zeros(32)
        v[:len(c["values"])] = c["values"]
        codes, sf = O.mx_quantize(v[None, :], 32)
        assert int(sf[0, 0]) == c["sf_byte"] == c["e"] + 127, c["name"]
        assert codes[0, :len(c["values"])].tolist() == [int(x, 16) for x in c["codes"]], c["name"]
        assert int(O.ue8m0_exponent(np.max(np.abs(v)))) == c["e"]


def test_mx_exponent_is_the_smallest_without_saturation_and_codes_are_nearest():
    rng = I._rng(12, 1)
    V = rng.standard_normal((40, 96)) * np.exp(rng.uniform(-20, 20, (40, 1)))
    V[3, 32:64] = 0
    V = V.astype(np.float32).astype(np.float64)
    codes, sf = O.mx_quantize(V, 32)
    assert codes.shape == V.shape and sf.shape == (40, 3) and sf.dtype == np.uint8
    e = sf.astype(np.int64) - 127
    amax = np.abs(V.reshape(40, 3, 32)).max(-1)
    nz = amax > 0
    assert np.all(amax[nz] <= 448.0 * np.ldexp(1.0, e[nz])) and np.all(amax[nz] > 448.0 * np.ldexp(1.0, e[nz] - 1))
    assert sf[3, 1] == 127 and np.all(codes[3, 32:64] & 0x7F == 0)
    # library pins: torch decodes the scale byte (float8_e8m0fnu) and casts the exactly scaled elements (float8_e4m3fn)
    s_t = torch.from_numpy(sf).view(torch.float8_e8m0fnu).to(torch.float64).numpy()
    assert np.array_equal(s_t, np.ldexp(1.0, e))
    q = torch.from_numpy(V.reshape(40, 3, 32) / s_t[..., None])
    assert np.array_equal(q.to(torch.float32).to(torch.float8_e4m3fn).view(torch.uint8).numpy().reshape(40, 96), codes)
    # dequantise: torch's decode of codes and scales == mx_dequantize; error <= half an e4m3 step of the block's scale
    deq_t = (torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy().reshape(40, 3, 32) * s_t[..., None])
    deq = O.mx_dequantize(codes, sf)
    assert np.array_equal(deq_t.reshape(40, 96), deq)
    step = np.repeat(np.ldexp(1.0, e), 32, axis=-1)
    assert np.all(np.abs(deq - V) <= 2.0 ** -4 * np.abs(V) + 2.0 ** -10 * step)
    # brute force nearest on a few blocks: no other code is closer
    t = O.e4m3_decode_table()[:0x7F]
    for r, b in ((0, 0), (7, 2), (39, 1)):
        for j in range(32):
            v = abs(V[r, b * 32 + j]) / 2.0 ** e[r, b]
            assert abs(t[codes[r, b * 32 + j] & 0x7F] - v) == np.min(np.abs(t - v))


def test_mx_scales_factor_out_per_block_and_block128_repeats():
    rng = I._rng(12, 2)
    V = rng.standard_normal((5, 256)).astype(np.float32).astype(np.float64)
    c0, s0 = O.mx_quantize(V, 32)
    V2 = V.copy()
    V2[:, 64:96] *= 2.0 ** 5                                   # scale ONE block by a power of two
    c1, s1 = O.mx_quantize(V2, 32)
    assert np.array_equal(c0, c1)
    d = s1.astype(int) - s0.astype(int)
    assert np.all(d[:, 2] == 5) and np.all(np.delete(d, 2, axis=1) == 0)
    # block 128: one exponent per 128 elements, stored four times; it is the max of the four 32-block exponents
    c128, s128 = O.mx_quantize(V2, 128)
    assert s128.shape == s1.shape
    grp = s1.reshape(5, 2, 4).max(-1)
    assert np.array_equal(s128.reshape(5, 2, 4), np.repeat(grp[..., None], 4, axis=-1))
    same = np.repeat(s128 == s1, 32, axis=-1)
    assert np.array_equal(c128[same], c1[same])                # blocks that kept their exponent keep their codes
    # a single block covering the whole row == the per-row recipe with a power-of-two scale
    r = V[:, :32]
    cr, sr = O.mx_quantize(r, 32)
    assert np.array_equal(cr, O.e4m3_encode(r / np.ldexp(1.0, sr.astype(int) - 127)))


def test_mx_layouts_of_the_weight_and_row_quantisers():
    d, f, E, R = 64, 96, 2, 6
    W = np.stack([I.make_expert_weight(1, e, d, f, 0.3 * (e + 1), 2) for e in range(E)])     # [E, K=d, N=f]
    codes, sf = O.mx_pack_weights(W)
    assert codes.shape == (E, f, d) and sf.shape == (E, f, d // 32)
    Wf = O.bf16_bits_to_f64(W)
    c_ref, s_ref = O.mx_quantize(Wf[1][:, 5][None, :], 32)     # feature 5 of expert 1: its K vector
    assert np.array_equal(codes[1, 5], c_ref[0]) and np.array_equal(sf[1, 5], s_ref[0])
    X = I.make_X(R, d, 3)
    xq, xs = O.mx_quantize_rows(X)
    assert xq.shape == (R, d) and xs.shape == (R, d // 32)
    assert np.array_equal(O.mx_quantize(O.bf16_bits_to_f64(X), 32)[0], xq)


def test_mx_ffn_reduces_to_the_plain_definition_and_tracks_the_bf16_ffn():
    """(i) On inputs that are exactly representable (e4m3 values times block scales) the block-scaled FFN is the
    plain SwiGLU FFN on the dequantised operands with one block quantisation of H: checked against an independent
    torch fp64 computation that decodes codes and scales with torch's own float8 types.  (ii) scales factor out:
    adding j to every scale byte of W2 multiplies Y by 2^j.  (iii) quantise -> MX FFN approximates the bf16 FFN,
    about as closely as the per-tensor recipe (on Gaussian data e4m3's 3 mantissa bits, not the scale granularity, set the error)."""
    cfg = I.scaled(I.C0, T=24, d=64, f=96, E=2, E_loc=2, k=1)
    L = I.make_layer(cfg, 4)
    ids = (np.arange(cfg.T) % 2).astype(np.int32)[:, None]
    off, r2a, a2r, Xp, R = O.permute(L["X"], ids, None, 2, 1)
    Y_ref, H_ref = O.grouped_ffn(Xp, off, r2a, L["W1"], L["W3"], L["W2"])
    W1q, W1s = O.mx_pack_weights(L["W1"]); W3q, W3s = O.mx_pack_weights(L["W3"]); W2q, W2s = O.mx_pack_weights(L["W2"])
    Xq, Xs = O.mx_quantize_rows(Xp)
    Y, Hq, Hs = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s)

    def deq(c, s):
        cv = torch.from_numpy(np.ascontiguousarray(c)).view(torch.float8_e4m3fn).to(torch.float64)
        sv = torch.from_numpy(np.ascontiguousarray(s)).view(torch.float8_e8m0fnu).to(torch.float64)
        return cv * sv.repeat_interleave(32, dim=-1)
    for e in range(2):
        rows = slice(int(off[e]), int(off[e + 1]))
        x = deq(Xq[rows], Xs[rows])
        h = torch.nn.functional.silu(x @ deq(W1q[e], W1s[e]).T) * (x @ deq(W3q[e], W3s[e]).T)
        hq, hs = O.mx_quantize(h.to(torch.float32).to(torch.float64).numpy(), 32)
        assert np.array_equal(hq, Hq[rows]) and np.array_equal(hs, Hs[rows])
        y = deq(Hq[rows], Hs[rows]) @ deq(W2q[e], W2s[e]).T
        assert np.allclose(Y[rows], y.numpy(), rtol=1e-12, atol=1e-300)
    Y2, _, _ = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s + np.uint8(3))
    assert np.allclose(Y2, 8.0 * Y, rtol=1e-15)
    # H_given: the down projection on given codes and scales -- the computed ones reproduce Y; one block's scale byte
    # raised by 1 doubles that block's contribution to its row (torch-decoded hand formula) and nothing else
    Yg, Hq2, Hs2 = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s, H_given=(Hq, Hs))
    assert np.array_equal(Yg, Y) and np.array_equal(Hq2, Hq) and np.array_equal(Hs2, Hs)
    r = int(off[1]) + 2
    Hs_alt = Hs.copy(); Hs_alt[r, 1] += 1
    Ya = O.grouped_ffn_mxfp8(Xq, Xs, off, r2a, W1q, W1s, W3q, W3s, W2q, W2s, H_given=(Hq, Hs_alt))[0]
    blk = deq(Hq[r:r + 1], Hs[r:r + 1])[:, 32:64] @ deq(W2q[1], W2s[1])[:, 32:64].T
    assert np.allclose(Ya[r] - Y[r], blk.numpy()[0], rtol=1e-9, atol=1e-12)
    others = np.ones(Y.shape[0], bool); others[r] = False
    assert np.array_equal(Ya[others], Y[others])
    m = O.ffn_error_metrics(Y, Y_ref)
    W1p, s1 = O.fp8_pack_weights(L["W1"]); W3p, s3 = O.fp8_pack_weights(L["W3"]); W2p, s2 = O.fp8_pack_weights(L["W2"])
    Xr, rs = O.fp8_quantize_rows(Xp)
    hsc = np.array([np.abs(H_ref[off[e]:off[e + 1]]).max() / 448.0 for e in range(2)], np.float32)
    Yt, _ = O.grouped_ffn_fp8(Xr, rs, off, r2a, W1p, s1, W3p, s3, W2p, s2, hsc)
    mt = O.ffn_error_metrics(Yt, Y_ref)
    assert m["mean_rel_err"] < 0.08 and m["max_abs_err_over_rms"] < 0.8, m
    assert m["mean_rel_err"] < 1.1 * mt["mean_rel_err"], (m, mt)
