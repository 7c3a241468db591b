"""Pins for the oracle's drift detector and incremental swap solver (O9, O10; f1) -- CPU only."""
import itertools
import json
import os

import numpy as np
import pytest
from scipy.spatial.distance import cosine as scipy_cosine

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import inputs as I

LIN = O.LatencyModel([1.0], [1.0])        # f(n) = n


# ---------------------------------------------------------------- O9 cosine distance
def test_cosine_distance_closed_forms_and_library():
    assert O.cosine_distance([1, 2, 3], [2, 4, 6]) == pytest.approx(0.0, abs=1e-15)      # parallel
    assert O.cosine_distance([1, 0, 0], [0, 5, 0]) == pytest.approx(1.0, abs=1e-15)      # orthogonal
    assert O.cosine_distance([1, 0], [1, 1]) == pytest.approx(1.0 - 2.0 ** -0.5, abs=1e-15)   # 45 degrees
    assert O.cosine_distance([3, 4], [4, 3]) == pytest.approx(1.0 - 24.0 / 25.0, abs=1e-15)
    assert O.cosine_distance([0, 0], [1, 2]) == 0.0 and O.cosine_distance([1, 2], [0, 0]) == 0.0   # D1
    rng = I._rng(3, 1)
    for _ in range(50):
        a, b = rng.uniform(0, 100, 256), rng.uniform(0, 100, 256)
        d = O.cosine_distance(a, b)
        assert d == pytest.approx(scipy_cosine(a, b), abs=1e-13)
        assert d == pytest.approx(O.cosine_distance(7.5 * a, 0.01 * b), abs=1e-13)       # scale invariance
        assert d == pytest.approx(O.cosine_distance(b, a), abs=1e-15)                    # symmetry
        assert 0.0 <= d <= 1.0                                                           # non-negative loads


# ---------------------------------------------------------------- O9 monitor (Alg. 1 phase 3)
def test_drift_monitor_cadence_threshold_and_cooldown():
    L, E, H, Wn = 2, 4, 10, 100
    a = np.array([[40.0, 30, 20, 10], [10, 10, 10, 10]])
    b = np.array([[10.0, 20, 30, 40], [10, 10, 10, 10]])      # layer 0 reverses, layer 1 unchanged
    m = O.DriftMonitor(L, E, window=Wn, H=H, delta=0.05)
    # no reference yet: never triggers, never checks
    for p in range(1, 101):
        trig, d = m.push(a)
        assert not trig and d is None
    m.set_reference(a)
    # steady state: checks on every H-th pass, distance 0
    for p in range(101, 121):
        trig, d = m.push(a)
        assert not trig
        assert (d is not None) == (p % H == 0)
        if d is not None:
            assert np.allclose(d, 0.0, atol=1e-15)
    # shift: after j shifted samples the window mean is ((Wn-j) a + j b)/Wn -> closed-form distance
    first = None
    for j in range(1, 101):
        p = 120 + j
        trig, d = m.push(b)
        w0 = ((Wn - j) * a[0] + j * b[0]) / Wn
        want = 1.0 - w0 @ a[0] / (np.linalg.norm(w0) * np.linalg.norm(a[0]))
        if p % H == 0:
            assert d[0] == pytest.approx(want, abs=1e-13) and d[1] == pytest.approx(0.0, abs=1e-15)
            assert trig == (want > 0.05)
            if trig and first is None:
                first = j
        else:
            assert d is None and not trig
    # independent computation of the first triggering pass: smallest multiple of H with d > delta
    js = [j for j in range(10, 101, 10)
          if 1.0 - (((Wn - j) * a[0] + j * b[0]) / Wn) @ a[0] /
          (np.linalg.norm(((Wn - j) * a[0] + j * b[0]) / Wn) * np.linalg.norm(a[0])) > 0.05]
    # by hand: j=30 -> w=(31,27,23,19), cos = 2700/sqrt(2580*3000) = 0.9705 (d = 0.029 < 0.05);
    #          j=40 -> w=(28,26,24,22), cos = 2600/sqrt(2520*3000) = 0.9456 (d = 0.054 > 0.05)
    assert first == js[0] == 40
    # rearrangement: reference := current window mean (all b by now), cooldown for H passes
    assert np.allclose(m.window_mean(), b)
    m.rearranged()
    assert np.allclose(m.ref, b)
    for i in range(H):
        trig, d = m.push(a)
        assert not trig and d is None            # suppressed, even on a multiple of H
    seen = 0
    for i in range(2 * H):
        trig, d = m.push(b)
        seen += d is not None
    assert seen == 2


# ---------------------------------------------------------------- O10 swap solver (Alg. 2)
def _direct_bin_latency(assign, load, G, scale, f, kind):
    """Independent statement of L_g (P:L182-L184 + M5): vectorised, no oracle code."""
    assign, load = np.asarray(assign), np.asarray(load, dtype=np.float64)
    if kind == O.MODEL_A:
        n = np.bincount(assign, weights=load, minlength=G)
        return np.array([f.whole_kernel(x) for x in n]) / np.asarray(scale)
    per = np.array([f.per_expert(x) for x in load])
    return np.bincount(assign, weights=per, minlength=G) / np.asarray(scale)


def _exhaustive_best_swap(assign, load, G, scale, f, kind):
    Lg = _direct_bin_latency(assign, load, G, scale, f, kind)
    hi, lo = int(np.argmax(Lg)), int(np.argmin(Lg))
    before = max(Lg[hi], Lg[lo])
    cands = []
    for ei, ej in itertools.product(np.flatnonzero(assign == hi), np.flatnonzero(assign == lo)):
        t = np.array(assign)
        t[ei], t[ej] = lo, hi
        Lt = _direct_bin_latency(t, load, G, scale, f, kind)
        cands.append((before - max(Lt[hi], Lt[lo]), -int(ei), -int(ej)))
    best = max(cands) if cands else (0.0, 0, 0)
    return best[0], (-best[1], -best[2]), Lg


def test_swap_refine_worked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "swap_refine_worked_example.json")))
    load, scale = np.array(g["load"], dtype=np.float64), g["scale"]
    assert np.allclose(O.bin_latencies(g["assign_start"], load, 2, scale, LIN, O.MODEL_A), g["start_bin_latency"])
    for key, c in g["candidate_swaps"].items():
        ei, ej = map(int, key.split(","))
        t = np.array(g["assign_start"])
        t[ei], t[ej] = t[ej], t[ei]
        Lt = O.bin_latencies(t, load, 2, scale, LIN, O.MODEL_A)
        assert np.allclose(Lt, c["bin_latency"])
        assert max(g["start_bin_latency"]) - Lt.max() == pytest.approx(c["reduction"])
    for kind in (O.MODEL_A, O.MODEL_B):       # identical for a linear f
        a, swaps = O.placement_swap_refine(g["assign_start"], load, 2, scale, LIN, kind, g["eps"])
        assert [list(s) for s in swaps] == g["swaps"] and a.tolist() == g["assign_final"]
        assert np.allclose(O.bin_latencies(a, load, 2, scale, LIN, kind), g["final_bin_latency"])
    n = g["no_reduction_case"]
    a, swaps = O.placement_swap_refine(n["assign_start"], n["load"], 2, n["scale"], LIN, O.MODEL_A, 0.03)
    assert swaps == [] and a.tolist() == n["assign_start"]


@pytest.mark.parametrize("kind", [O.MODEL_A, O.MODEL_B])
@pytest.mark.parametrize("E,G,seed", [(8, 2, 0), (12, 3, 1), (16, 4, 2), (24, 4, 3), (32, 8, 4)])
def test_swap_refine_invariants_and_exhaustive_steps(E, G, seed, kind):
    rng = I._rng(seed, 77)
    load = np.floor(rng.pareto(1.2, E) * 40 + 1)
    scale = I.make_throughput_scales(G, seed)
    f = O.LatencyModel([1, 16, 64, 256, 1024], [5.0, 5.5, 7.0, 19.0, 75.0], E_prof=E // G)   # floor + linear tail
    start = O.placement_contiguous(E, G)
    a, swaps = O.placement_swap_refine(start, load, G, scale, f, kind, 0.03)
    # replay: every applied swap is the exhaustive best one, the max never increases, counts are kept
    cur = np.array(start)
    prev_max = _direct_bin_latency(cur, load, G, scale, f, kind).max()
    for (ei, ej) in swaps:
        red, best, Lg = _exhaustive_best_swap(cur, load, G, scale, f, kind)
        assert Lg.max() > 1.03 * Lg.mean() and red > 0 and best == (ei, ej)
        assert cur[ei] == int(np.argmax(Lg)) and cur[ej] == int(np.argmin(Lg))
        cur[ei], cur[ej] = cur[ej], cur[ei]
        now = _direct_bin_latency(cur, load, G, scale, f, kind).max()
        assert now <= prev_max + 1e-12
        prev_max = now
    assert np.array_equal(cur, a)
    assert np.array_equal(np.bincount(a, minlength=G), np.bincount(start, minlength=G))
    # termination: stop rule met, or no swap between slowest and fastest reduces the pair's max
    red, _, Lg = _exhaustive_best_swap(a, load, G, scale, f, kind)
    assert Lg.max() <= 1.03 * Lg.mean() or red <= 0
    assert Lg.max() <= _direct_bin_latency(start, load, G, scale, f, kind).max() + 1e-12
    # max_swaps is respected and is a prefix of the unbounded run
    if swaps:
        a1, s1 = O.placement_swap_refine(start, load, G, scale, f, kind, 0.03, max_swaps=1)
        assert s1 == swaps[:1]
    # eps large enough => nothing to do
    a2, s2 = O.placement_swap_refine(start, load, G, scale, f, kind, eps=1e9)
    assert s2 == [] and np.array_equal(a2, start)
