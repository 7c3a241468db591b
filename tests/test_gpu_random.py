"""Seeded random configurations through the C ABI against the oracle -- a fixed slice of the randomised comparison
described in DESIGN.md section 4 (which ran hundreds of thousands of cases once): route over every score / group /
renormalisation combination and nine logit families, permute over random shapes and expert maps, the whole layer over the
three config families.  Integer outputs bit-exact, gate weights to 1e-6, `out` inside its derived bound on sampled tokens."""
import numpy as np
import pytest
import torch

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import binding as B
from paper_2606_00735_b200 import inputs as I
from test_gpu_parity import W_RTOL, check_layer_output, check_permute, dev, host_bits, layer_device_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    B.load()
    torch.cuda.set_device(0)


def _logits(rng, T, E):
    kind = int(rng.integers(0, 9))
    x = rng.standard_normal((T, E)).astype(np.float32) * np.float32(rng.choice([0.01, 0.3, 1.0, 4.0, 30.0]))
    if kind == 1:
        x = x.astype(np.float16).astype(np.float32)                                        # fp16-valued
    elif kind == 2:
        x = (x.view(np.uint32) & np.uint32(0xffff0000)).view(np.float32)                   # bf16-valued: exact ties
    elif kind == 3:
        x = np.round(x * 4) / 4
    elif kind == 4:                                                                        # keys a few ulps apart
        base = rng.standard_normal((T, 1)).astype(np.float32)
        x = (np.broadcast_to(base, (T, E)).copy().view(np.int32) + rng.integers(-300, 300, (T, E), dtype=np.int32)).view(np.float32)
    elif kind == 5:                                                                        # masked experts
        x[rng.random((T, E)) < rng.choice([0.5, 0.9, 0.98])] = -np.inf
        x[:, :min(E, 4)] = rng.standard_normal((T, min(E, 4))).astype(np.float32)
    elif kind == 6:                                                                        # signed zeros
        x = np.where(rng.random((T, E)) < 0.5, np.float32(0.0), np.float32(-0.0)) + (rng.random((T, E)) < 0.05) * x
    elif kind == 7:
        x = (x * 1e-30).astype(np.float32)                                                 # towards the denormals
    elif kind == 8:                                                                        # one lane holds the top
        v = max(1, E // 8)
        lane = int(rng.integers(0, 8))
        x[:, lane * v:(lane + 1) * v] += np.float32(rng.choice([0.5, 3.0, 20.0]))
    return np.ascontiguousarray(x.astype(np.float32)), kind


@pytest.mark.parametrize("seed", range(8))
def test_route_random_configs(seed):
    rng = np.random.default_rng(1000 + seed)
    for case in range(25):
        wide = rng.random() < 0.6
        E = int(rng.choice([128, 256])) if wide else int(rng.choice([8, 16, 32, 33, 64, 96, 160, 384, 512]))
        k = int(rng.integers(1, 9)) if wide or rng.random() < 0.7 else int(rng.integers(1, min(E, 32) + 1))
        k = min(k, E)
        T = int(rng.choice([1, 3, 4, 5, 37, 300, 1027, 4099]))
        sf = int(rng.integers(0, 2))
        divs = [g for g in (2, 3, 4, 5, 8, 16) if E % g == 0]
        ng = int(rng.choice([0, 8])) if wide else (int(rng.choice(divs)) if divs and rng.random() < 0.5 else 0)
        tg = int(rng.integers(1, ng + 1)) if ng else 0
        if ng and tg * (E // ng) < k:
            tg = ng
        renorm = 1 if not sf else int(rng.integers(0, 2))
        if not sf and rng.random() < 0.15:
            renorm = 0
        x, kind = _logits(rng, T, E)
        bias = None
        if sf and rng.random() < 0.7:
            bias = (rng.standard_normal(E) * rng.choice([0.01, 0.3, 3.0])).astype(np.float32)
        kw = dict(num_experts=E, top_k=k, score_fn=sf, renormalize=renorm, routed_scale=float(rng.choice([1.0, 2.5])),
                  n_group=ng, topk_group=tg)
        with np.errstate(all="ignore"):                    # masked rows: 0 / 0 weights on both sides
            ids_o, w_o, c_o = O.route_topk(x, select_bias=bias, **kw)
        rc = B.RouteConfig(select_bias=dev(bias) if bias is not None else None, **kw)
        ids, w, cnt = B.route_topk(dev(x), rc)
        torch.cuda.synchronize()
        tag = (seed, case, kw, T, kind)
        assert np.array_equal(ids.cpu().numpy(), ids_o), tag
        assert np.array_equal(cnt.cpu().numpy(), c_o), tag
        wg = w.cpu().numpy().astype(np.float64)
        ok = np.isfinite(w_o) & (np.abs(w_o) > 1e-30)      # (below: f32 denormals, where one ulp is a large relative step)
        if ok.any():
            assert np.max(np.abs(wg[ok] - w_o[ok]) / np.abs(w_o[ok])) <= W_RTOL, tag


@pytest.mark.parametrize("seed", range(3))
def test_permute_random_shapes(seed):
    rng = np.random.default_rng(2000 + seed)
    for case in range(12):
        E = int(rng.choice([1, 2, 8, 33, 64, 128, 256, 300, 1024]))
        k = int(rng.integers(1, min(E, 8) + 1))
        T = int(rng.choice([1, 2, 31, 257, 1000, 4097, 20000]))
        d = int(rng.choice([8, 64, 136, 1024]))
        if T * d > 8e6:
            d = 64
        align = int(rng.choice([1, 8, 16, 64, 128]))
        ids = np.argsort(rng.random((T, E)), axis=1)[:, :k].astype(np.int32)
        if rng.random() < 0.2:
            ids[:] = ids[0]                                                   # every token to the same experts
        if rng.integers(0, 3) == 0 or E == 1:
            emap, E_loc = None, E
        else:
            E_loc = int(rng.integers(1, E + 1))
            emap = np.full(E, -1, np.int32)
            emap[rng.permutation(E)[:E_loc]] = rng.permutation(E_loc).astype(np.int32)
        check_permute(I.make_X(T, d, int(rng.integers(0, 1000))), ids, emap, E, E_loc, align)


@pytest.mark.parametrize("seed", range(3))
def test_layer_random_configs(seed):
    rng = np.random.default_rng(3000 + seed)
    for case in range(8):
        base = [I.C1, I.C2, I.C3][int(rng.integers(0, 3))]
        E = int(rng.choice([8, 16, 64, 128, 256])) if base is not I.C3 else int(rng.choice([64, 128, 256]))
        E_loc = E if rng.random() < 0.5 else max(1, E // int(rng.choice([2, 4, 8, 32])))
        k = int(rng.integers(1, min(8, E) + 1))
        if base is I.C3:
            k = min(k, 4 * (E // 8))
        T = int(rng.choice([1, 2, 5, 63, 64, 65, 300, 1000, 2500]))
        d, f = int(rng.choice([64, 128, 256, 512])), int(rng.choice([64, 128, 320, 512]))
        cfg = I.scaled(base, T=T, d=d, f=f, E=E, E_loc=E_loc, k=k)
        policy = str(rng.choice(["contiguous", "random"])) if E_loc < E else "contiguous"
        L = I.make_layer(cfg, int(rng.integers(0, 1000)), map_policy=policy)
        rc, lg, X, emap, W1, W3, W2 = layer_device_inputs(cfg, L)
        out, counts = B.moe_layer_forward(rc, lg, X, emap, W1, W3, W2)
        torch.cuda.synchronize()
        ids, w, c = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
        tag = (seed, case, base.name, T, k, E, E_loc, d, f, policy)
        assert np.array_equal(counts.cpu().numpy(), c), tag
        em = L["expert_map"] if E_loc < E else None
        slot = ids if em is None else em[ids]
        res = np.nonzero((slot >= 0).any(axis=1))[0]
        if len(res):
            sample = sorted(set(rng.choice(res, size=min(6, len(res)), replace=False).tolist() + [int(res[0]), int(res[-1])]))
            ref, ref_abs = O.moe_layer_direct(L["X"], ids, w, em, L["W1"], L["W3"], L["W2"], tokens=sample, return_abs=True)
            got = O.bf16_bits_to_f64(host_bits(out[sample]))
            check_layer_output(got, np.stack([ref[t] for t in sample]), np.stack([ref_abs[t] for t in sample]))
        none = np.nonzero(~(slot >= 0).any(axis=1))[0]
        if len(none):
            assert torch.count_nonzero(out[torch.from_numpy(none[:256]).cuda()].view(torch.int16)).item() == 0, tag


@pytest.mark.parametrize("seed", range(2))
def test_fp8_ffn_random_ragged_segments(seed):
    """Both FP8 kinds on random ragged segment lists around the tile boundaries (the bodies of the fixed ragged tests:
    H codes within one step, GEMM-2 on the device's own codes element by element, Y at the stated bars)."""
    from test_gpu_mxfp8 import test_ffn_mxfp8_ragged_token_tiles
    from test_gpu_parity import test_ffn_fp8_ragged_token_tiles
    rng = np.random.default_rng(4000 + seed)
    pool = [0, 1, 15, 16, 17, 31, 33, 63, 64, 65, 127, 128, 129, 191, 192, 193, 255, 256, 257, 383, 385, 511, 513, 769]
    for case in range(4):
        E = int(rng.choice([2, 3, 5, 8]))
        rows = [int(x) for x in rng.choice(pool, E)]
        if sum(rows) == 0:
            rows[0] = 40
        d, f = int(rng.choice([128, 256, 384])), int(rng.choice([128, 256, 640]))
        test_ffn_fp8_ragged_token_tiles(rows, d, f)
        test_ffn_mxfp8_ragged_token_tiles(rows, d, f)
