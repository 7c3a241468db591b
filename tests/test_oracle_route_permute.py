"""Pins for the oracle's route / histogram / permute (O1, O2) -- CPU only.

Each test pins the oracle to something other than itself: brute-force sorting,
closed forms, scipy library routines, np.argsort(kind='stable'), or hand-worked
golden fixtures (tests/golden/*.json, each with its citation)."""
import json
import os

import numpy as np
import pytest
import scipy.special

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import inputs as I


def brute_topk(keys, k):
    """Sort all E keys by (-key, index) in pure Python."""
    out = []
    for row in keys:
        order = sorted(range(len(row)), key=lambda e: (-float(row[e]), e))
        out.append(order[:k])
    return np.array(out, dtype=np.int32)


# ---------------------------------------------------------------- a1 ids
@pytest.mark.parametrize("E,k,seed", [(8, 2, 0), (128, 8, 1), (33, 5, 2), (256, 8, 3)])
def test_softmax_ids_match_brute_force_sort(E, k, seed):
    z = I.make_logits(97, E, 1.2, seed)
    ids, w, counts = O.route_topk(z, E, k)
    assert np.array_equal(ids, brute_topk(z, k))


def test_softmax_then_topk_ids_equal_topk_of_probabilities():
    z = I.make_logits(64, 16, 0.7, 5)
    ids, _, _ = O.route_topk(z, 16, 4)
    p = scipy.special.softmax(z.astype(np.float64), axis=1)
    assert np.array_equal(ids, brute_topk(p, 4))


def test_adversarial_ties():
    E, k = 16, 4
    allsame = np.full((3, E), 0.25, np.float32)
    ids, w, c = O.route_topk(allsame, E, k)
    assert np.array_equal(ids, np.tile(np.arange(k), (3, 1)))
    assert np.allclose(w, 0.25, atol=0, rtol=1e-7)
    # duplicated maxima: lowest index first
    z = np.zeros((1, E), np.float32)
    z[0, [3, 9, 12]] = 7.0
    z[0, 5] = 6.0
    ids, _, _ = O.route_topk(z, E, k)
    assert ids.tolist() == [[3, 9, 12, 5]]
    # one-hot
    z = np.full((1, E), -3.0, np.float32)
    z[0, 11] = 9.0
    ids, _, _ = O.route_topk(z, E, 1)
    assert ids.tolist() == [[11]]
    # +0.0 and -0.0 compare equal -> lower index wins
    z = np.full((1, E), -1.0, np.float32)
    z[0, 2] = -0.0
    z[0, 7] = 0.0
    ids, _, _ = O.route_topk(z, E, 2)
    assert ids.tolist() == [[2, 7]]
    # k == E: a permutation sorted by (-key, idx)
    z = I.make_logits(5, E, 0.0, 9)
    ids, w, c = O.route_topk(z, E, E, renormalize=0)
    assert np.array_equal(np.sort(ids, axis=1), np.tile(np.arange(E), (5, 1)))
    # k == E, no renorm => the full softmax (library routine)
    p = scipy.special.softmax(z.astype(np.float64), axis=1)
    assert np.allclose(w, np.take_along_axis(p, ids.astype(np.int64), 1), rtol=2e-7, atol=0)


def test_group_limited_golden(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "group_limited_example.json")))
    z = np.array(g["logits"], np.float32)
    ids, w, c = O.route_topk(z, g["E"], g["k"], n_group=g["n_group"], topk_group=g["topk_group"])
    assert ids.tolist() == g["ids"]


@pytest.mark.parametrize("score_fn", [O.SCORE_SOFTMAX, O.SCORE_SIGMOID])
def test_group_limited_degenerate_cases_equal_ungrouped(score_fn):
    E, k = 64, 6
    z = I.make_logits(200, E, 1.0, 4)
    b = I.make_select_bias(E, 4) if score_fn == O.SCORE_SIGMOID else None
    base = O.route_topk(z, E, k, score_fn=score_fn, select_bias=b)
    one_group = O.route_topk(z, E, k, score_fn=score_fn, select_bias=b, n_group=1, topk_group=1)
    all_groups = O.route_topk(z, E, k, score_fn=score_fn, select_bias=b, n_group=8, topk_group=8)
    for other in (one_group, all_groups):
        assert np.array_equal(base[0], other[0])
        assert np.array_equal(base[1], other[1])
        assert np.array_equal(base[2], other[2])


def test_group_limited_brute_force_sigmoid():
    """Independent re-derivation of steps 2-4 with python loops on a small case."""
    E, k, ng, tg = 32, 4, 8, 3
    z = I.make_logits(50, E, 1.2, 6)
    b = I.make_select_bias(E, 6)
    ids, w, c = O.route_topk(z, E, k, score_fn=O.SCORE_SIGMOID, select_bias=b, n_group=ng, topk_group=tg)
    key = (O.vsig_f32(z) + b[None, :]).astype(np.float32)
    gs = E // ng
    for t in range(z.shape[0]):
        scores = []
        for g in range(ng):
            vals = sorted((float(v) for v in key[t, g * gs:(g + 1) * gs]), reverse=True)
            scores.append(float(np.float32(np.float32(vals[0]) + np.float32(vals[1]))))
        kept = sorted(range(ng), key=lambda g: (-scores[g], g))[:tg]
        cand = [e for e in range(E) if e // gs in kept]
        order = sorted(cand, key=lambda e: (-float(key[t, e]), e))[:k]
        assert ids[t].tolist() == order
        assert all(e // gs in kept for e in ids[t])


def test_fewer_than_k_finite_keys_still_gives_k_distinct_experts():
    """R3 with keys of -inf (masked logits; a group limit that leaves fewer than k finite keys): the picks are the
    first k of the order (key descending, index ascending) -- k DISTINCT experts -- and the kept groups are the first
    topk_group of (score descending, group ascending).  Pinned against a pure-Python sort, with hand-worked rows."""
    E, k = 16, 5
    z = np.full((3, E), -np.inf, np.float32)
    z[0, [9, 3]] = [1.0, 2.0]                     # two finite keys: 3, 9, then the lowest unpicked indices 0, 1, 2
    z[1, :] = -np.inf                             # none finite: 0, 1, 2, 3, 4
    z[2, [0, 1, 2, 15]] = [0.5, 0.5, -1.0, 7.0]   # 15, 0, 1, 2, then 3
    with np.errstate(invalid="ignore"):          # the all -inf row has no defined weights (NaN): ids only
        ids, _, counts = O.route_topk(z, E, k, renormalize=0)
    assert ids.tolist() == [[3, 9, 0, 1, 2], [0, 1, 2, 3, 4], [15, 0, 1, 2, 3]]
    assert counts.sum() == 3 * k and all(len(set(r)) == k for r in ids.tolist())
    rng = np.random.default_rng(5)
    zz = rng.standard_normal((200, 32)).astype(np.float32)
    zz[rng.random(zz.shape) < 0.85] = -np.inf
    assert np.array_equal(O.route_topk(zz, 32, 8, renormalize=0)[0], brute_topk(zz, 8))
    # groups: 4 groups of 8; scores of -inf tie and go to the lower group index; all groups kept when topk_group = 4
    ng, tg, gs = 4, 2, 8
    for tg in (1, 2, 4):
        ids, _, _ = O.route_topk(zz, 32, 8, renormalize=0, n_group=ng, topk_group=tg)
        for t in range(zz.shape[0]):
            scores = []
            for g in range(ng):
                vals = sorted((float(v) for v in zz[t, g * gs:(g + 1) * gs]), reverse=True)
                scores.append(float(np.float32(vals[0]) + np.float32(vals[1])))
            kept = sorted(range(ng), key=lambda g: (-scores[g], g))[:tg]
            keyt = [float(zz[t, e]) if e // gs in kept else -np.inf for e in range(32)]
            order = sorted(range(32), key=lambda e: (-keyt[e], e))[:8]
            assert ids[t].tolist() == order, (tg, t)


# ---------------------------------------------------------------- vsig (selection key)
def test_vsig_accuracy_monotone_and_closed_forms():
    xs = np.concatenate([np.linspace(-30, 30, 200001), I._rng(0, 1).standard_normal(100000) * 3]).astype(np.float32)
    v = O.vsig_f32(xs)
    assert v.dtype == np.float32
    ref = scipy.special.expit(xs.astype(np.float64))
    rel = np.abs(v.astype(np.float64) - ref) / ref
    assert rel.max() < 4e-7, rel.max()
    # closed forms
    assert O.vsig_f32(np.float32(0.0)) == np.float32(0.5)
    assert np.all(O.vsig_f32(np.array([100.0, 80.0], np.float32)) == np.float32(1.0))
    tiny = O.vsig_f32(np.array([-100.0, -80.0], np.float32))
    assert tiny[0] == tiny[1] and 0 < tiny[0] < 1e-34
    # symmetry s(x)+s(-x)=1 within rounding
    xs2 = np.linspace(-12, 12, 4001).astype(np.float32)
    assert np.max(np.abs(O.vsig_f32(xs2).astype(np.float64) + O.vsig_f32(-xs2) - 1.0)) < 3e-7
    # weakly monotone on a sorted grid up to 1 ulp wiggle: selection needs a well-defined key,
    # not strict monotonicity; check no inversion larger than 2 ulp
    srt = np.sort(xs)
    vs = O.vsig_f32(srt).astype(np.float64)
    inv = np.maximum(0.0, vs[:-1] - vs[1:]) / np.maximum(vs[1:], 1e-300)
    assert inv.max() < 2.5e-7


def test_vsig_has_no_fma_dependence():
    """The definition is a sequence of separately rounded binary32 ops; emulate each op
    in f64-then-round (exact for +,-,* of two f32) and demand bit equality."""
    f = np.float32
    xs = I._rng(7, 1).standard_normal(5000).astype(np.float32) * 4
    got = O.vsig_f32(xs)
    for x, gv in zip(xs[:1500], got[:1500]):
        x = f(min(max(x, f(-80)), f(80)))
        a = f(-x)
        n = f(np.rint(f(np.float64(a) * np.float64(O._LOG2E))))
        r = f(np.float64(a) - np.float64(f(np.float64(n) * np.float64(O._LN2_HI))))
        r = f(np.float64(r) - np.float64(f(np.float64(n) * np.float64(O._LN2_LO))))
        p = O._VSIG_COEF[0]
        for c in O._VSIG_COEF[1:]:
            p = f(np.float64(p) * np.float64(r))
            p = f(np.float64(p) + np.float64(c))
        e = f(np.ldexp(np.float64(p), int(n)))
        den = f(np.float64(1.0) + np.float64(e))
        want = f(1.0) / den          # numpy scalar f32 division: IEEE binary32
        assert want == gv


# ---------------------------------------------------------------- a1 weights
@pytest.mark.parametrize("E,k", [(8, 2), (128, 8)])
def test_softmax_renorm_equals_softmax_over_selected(E, k):
    z = I.make_logits(300, E, 1.0, 11)
    ids, w, _ = O.route_topk(z, E, k, renormalize=1)
    sel = np.take_along_axis(z.astype(np.float64), ids.astype(np.int64), 1)
    want = scipy.special.softmax(sel, axis=1)
    assert np.max(np.abs(w - want) / want) < 1.5e-7          # one f32 rounding
    assert np.max(np.abs(w.astype(np.float64).sum(1) - 1.0)) < 4 * 2 ** -23
    ids2, w2, _ = O.route_topk(z, E, k, renormalize=0)
    assert np.array_equal(ids, ids2)
    assert np.all(w2.astype(np.float64).sum(1) <= 1.0 + 1e-6)
    full = scipy.special.softmax(z.astype(np.float64), axis=1)
    assert np.allclose(w2, np.take_along_axis(full, ids.astype(np.int64), 1), rtol=1.5e-7, atol=0)


def test_sigmoid_weights_exclude_bias_and_scale():
    E, k = 64, 8
    z = I.make_logits(100, E, 1.2, 12)
    b = I.make_select_bias(E, 12) * 50          # large bias: selection changes, weights must not include it
    ids, w, _ = O.route_topk(z, E, k, score_fn=O.SCORE_SIGMOID, select_bias=b, renormalize=0)
    s = scipy.special.expit(np.take_along_axis(z.astype(np.float64), ids.astype(np.int64), 1))
    assert np.max(np.abs(w - s) / s) < 1.5e-7
    ids_nb, _, _ = O.route_topk(z, E, k, score_fn=O.SCORE_SIGMOID, renormalize=0)
    assert not np.array_equal(ids, ids_nb)
    _, w25, _ = O.route_topk(z, E, k, score_fn=O.SCORE_SIGMOID, select_bias=b, renormalize=1, routed_scale=2.5)
    assert np.allclose(w25.astype(np.float64).sum(1), 2.5, rtol=1e-6)
    sn = s / s.sum(1, keepdims=True) * 2.5
    assert np.max(np.abs(w25 - sn) / sn) < 1.5e-7


# ---------------------------------------------------------------- a2 histogram
def test_histogram_invariants():
    cfg = I.C2
    z = I.make_logits(1024, cfg.E, cfg.zipf_s, 0)
    ids, _, counts = O.route_topk(z, cfg.E, cfg.k)
    assert counts.sum() == 1024 * cfg.k
    assert np.array_equal(counts, np.bincount(ids.ravel(), minlength=cfg.E))
    parts = sum(O.route_topk(z[i:i + 256], cfg.E, cfg.k)[2] for i in range(0, 1024, 256))
    assert np.array_equal(parts, counts)
    # every token's ids are distinct
    assert all(len(set(r)) == cfg.k for r in ids.tolist())


# ---------------------------------------------------------------- a3 permute
def _check_permute(X, ids, emap, E_loc, align):
    T, k = ids.shape
    off, r2a, a2r, Xp, R = O.permute(X, ids, emap, E_loc, align)
    E = len(emap) if emap is not None else E_loc
    m = np.arange(E) if emap is None else emap
    slot = m[ids.reshape(-1)]
    cnt = np.bincount(slot[slot >= 0], minlength=E_loc)
    assert np.array_equal(np.diff(off), (cnt + align - 1) // align * align)
    assert R == cnt.sum()
    real = np.nonzero(r2a >= 0)[0]
    assert len(real) == R
    # bijection onto resident assignments
    assert np.array_equal(a2r[r2a[real]], real)
    assert np.array_equal(np.sort(r2a[real]), np.nonzero(slot >= 0)[0])
    assert np.all(a2r[slot < 0] == -1)
    for s in range(E_loc):
        seg = r2a[off[s]:off[s + 1]]
        segr = seg[seg >= 0]
        assert len(segr) == cnt[s] and np.all(seg[cnt[s]:] == -1)       # padding at the end
        assert np.all(np.diff(segr) > 0)                                  # stability
        assert np.all(slot[segr] == s)
    assert np.array_equal(Xp[real], X[r2a[real] // k])                   # bitwise row copies
    assert np.all(Xp[r2a < 0] == 0)
    # library pin: stable argsort by slot
    order = np.argsort(np.where(slot >= 0, slot, E_loc + 1), kind="stable")[:R]
    if align == 1:
        assert np.array_equal(r2a, order)
    return off, r2a, a2r, Xp


@pytest.mark.parametrize("align", [1, 8, 128])
def test_permute_identity_map(align):
    cfg = I.C0
    L = I.make_layer(cfg, 0, with_weights=False)
    ids, _, _ = O.route_topk(L["logits"], cfg.E, cfg.k)
    off, r2a, a2r, Xp = _check_permute(L["X"], ids, None, cfg.E, align)
    if align == 1:
        assert off[-1] == cfg.T * cfg.k


@pytest.mark.parametrize("policy", ["contiguous", "strided", "random"])
def test_permute_partial_residency(policy):
    cfg = I.scaled(I.C3, T=257, d=64)
    L = I.make_layer(cfg, 3, with_weights=False, map_policy=policy)
    ids, _, _ = O.route_topk(L["logits"], select_bias=L["select_bias"], **I.route_kwargs(cfg))
    _check_permute(L["X"], ids, L["expert_map"], cfg.E_loc, 1)
    _check_permute(L["X"], ids, L["expert_map"], cfg.E_loc, 16)


def test_permute_empty_experts_and_no_resident():
    X = I.make_X(4, 16, 0)
    ids = np.array([[5, 6], [5, 7], [6, 5], [7, 6]], np.int32)
    emap = np.full(8, -1, np.int32)
    emap[5] = 1          # slots 0 and 2 empty
    off, r2a, a2r, Xp, R = O.permute(X, ids, emap, 3, 1)
    assert off.tolist() == [0, 0, 3, 3] and R == 3
    assert r2a.tolist() == [0, 2, 5]
    assert a2r.tolist() == [0, -1, 1, -1, -1, 2, -1, -1]
    emap[:] = -1
    off, r2a, a2r, Xp, R = O.permute(X, ids, emap, 3, 1)
    assert off.tolist() == [0, 0, 0, 0] and R == 0 and len(r2a) == 0 and np.all(a2r == -1)
