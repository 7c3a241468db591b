"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/vibe.h
declares, rejects bad arguments before touching CUDA, and its HOST-side placement code
(a7/a8) agrees with the oracle.  No GPU compute is called here."""
import itertools
import json
import os
import re

import numpy as np
import pytest

from oracle import vibe_oracle as O
from paper_2606_00735_b200 import binding as B
from paper_2606_00735_b200 import build as build_mod
from paper_2606_00735_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build()
    return B.load()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "vibe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"VIBE_API\s+[\w\s\*]+?\b(vibe_\w+)\s*\(", hdr))
    assert declared == set(B.EXPORTED_SYMBOLS), declared ^ set(B.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.vibe_version() >= 100
    assert lib.vibe_status_string(0) == b"VIBE_OK"
    assert lib.vibe_status_string(4) == b"VIBE_ERR_CUDA"


def test_argument_errors_are_detected_before_any_launch(lib):
    import ctypes as C
    cfg = B._RouteCfg(8, 9, 0, 1, 1.0, 0, 0, None)                 # k > E
    assert lib.vibe_route_topk(C.byref(cfg), None, 4, None, None, None, None) == 1
    assert b"k <= E" in lib.vibe_last_error()
    cfg = B._RouteCfg(8, 2, 7, 1, 1.0, 0, 0, None)                 # bad score_fn
    assert lib.vibe_route_topk(C.byref(cfg), None, 4, None, None, None, None) == 1
    cfg = B._RouteCfg(256, 8, 1, 1, 1.0, 7, 4, None)               # E % n_group
    assert lib.vibe_route_topk(C.byref(cfg), None, 4, None, None, 1, None) == 1
    cfg = B._RouteCfg(256, 8, 1, 1, 1.0, 64, 1, None)              # topk_group*gs < k
    assert lib.vibe_route_topk(C.byref(cfg), None, 4, None, None, 1, None) == 1
    cfg = B._RouteCfg(1024, 8, 0, 1, 1.0, 0, 0, None)              # unsupported E
    assert lib.vibe_route_topk(C.byref(cfg), 16, 4, 16, 16, 16, None) == 2
    # permute: d % 8, NULL map with E_loc != E, short workspace
    assert lib.vibe_permute(16, 16, None, None, 4, 12, 2, 8, 8, 1, 16, 16, 16, 16, 16, 1 << 20, None) == 1
    assert lib.vibe_permute(16, 16, None, None, 4, 16, 2, 8, 4, 1, 16, 16, 16, 16, 16, 1 << 20, None) == 1
    assert lib.vibe_permute(16, 16, None, None, 4, 16, 2, 8, 8, 1, 16, 16, 16, 16, 16, 8, None) == 3
    # permute without a workspace argument: bad sizes; more slots than the static scratch array holds (no launch either way)
    assert lib.vibe_permute_static(16, 16, None, None, -1, 16, 2, 8, 8, 1, 16, 16, 16, 16, None) == 1
    assert lib.vibe_permute_static(16, 16, None, None, 4, 16, 2, 2048, 1024, 1, 16, 16, 16, 16, None) == 3
    assert b"static array" in lib.vibe_last_error()
    # ffn: shape limits, misalignment
    assert lib.vibe_grouped_ffn(16, 16, 8, 64, 100, 128, 16, 16, 16, 16, 16, None, 0, None) == 2
    assert lib.vibe_grouped_ffn(8, 16, 8, 64, 128, 128, 16, 16, 16, 16, 16, None, 0, None) == 1
    assert lib.vibe_combine(16, 16, 16, 4, 2, 12, 16, None) == 1
    assert lib.vibe_combine(16, 16, 16, 4, 64, 16, 16, None) == 2


def test_workspace_sizes(lib):
    assert B.rows_cap(64, 2, 8, 1) == 128
    assert B.rows_cap(64, 8, 4, 1) == 64 * 4
    assert B.rows_cap(64, 2, 8, 128) == 128 + 8 * 127
    assert B.workspace_bytes(B.WS_PERMUTE, 64, 2, 8, 8, 256, 512) >= 8 * 4 * 2
    lay = B.workspace_bytes(B.WS_LAYER, 64, 2, 8, 8, 256, 512)
    assert lay >= 128 * (256 * 2 * 2 + 512 * 2)
    assert B.workspace_bytes(B.WS_LAYER_HOST, 64, 2, 8, 8, 256, 512) > lay
    assert B.workspace_bytes(99, 64, 2, 8, 8, 256, 512) == 0


# ------------------------------------------------------------------ placement (host code) vs oracle
def _models():
    return [
        (None, O.LatencyModel([1.0], [1.0])),
        (B.LatencyModel([1, 8, 64, 256, 1024], [12.0, 12.5, 11.0, 30.0, 110.0], 4),
         O.LatencyModel([1, 8, 64, 256, 1024], [12.0, 12.5, 11.0, 30.0, 110.0], 4)),
    ]


def test_placement_worked_example_through_the_abi(lib, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "placement_worked_example.json")))
    a = B.placement_greedy(g["load"], 2, g["scale"], None)
    assert a.tolist() == g["greedy_assign"]
    sc, per = B.placement_eval(a, g["load"], 2, g["scale"], None, B.MODEL_A)
    assert sc == pytest.approx(g["greedy_score"], rel=1e-12)
    assert per.tolist() == pytest.approx([19.0, 20.0], rel=1e-12)
    tb = B.placement_token_balanced(g["load"], 2)
    assert tb.tolist() == g["token_balanced_assign"]
    assert B.placement_eval(tb, g["load"], 2, g["scale"], None)[0] == pytest.approx(g["token_balanced_score"], rel=1e-12)
    assert B.placement_contiguous(8, 2).tolist() == [0, 0, 0, 0, 1, 1, 1, 1]


@pytest.mark.parametrize("G,E", [(2, 8), (3, 7), (4, 6)])
def test_placement_eval_matches_oracle_on_every_binning(lib, G, E):
    rng = I._rng(40 + G, E)
    load = rng.integers(0, 1500, E).astype(np.float64)
    scale = I.make_throughput_scales(G, 9)
    for bm, om in _models():
        for kind in (B.MODEL_A, B.MODEL_B):
            best = np.inf
            for a in itertools.product(range(G), repeat=E):
                got, per = B.placement_eval(a, load, G, scale, bm, kind)
                want, wper = O.placement_eval(a, load, G, scale, om, kind)
                assert got == pytest.approx(want, rel=1e-12)
                assert per == pytest.approx(wper, rel=1e-12)
                best = min(best, got)
            gr = B.placement_greedy(load, G, scale, bm)
            assert np.array_equal(gr, O.placement_greedy(load, G, scale, om))
            assert B.placement_eval(gr, load, G, scale, bm, kind)[0] >= best * (1 - 1e-12)


@pytest.mark.parametrize("s,T", [(0.8, 2048), (1.2, 16384), (1.6, 2048)])
def test_placement_stress_shapes_match_oracle(lib, s, T):
    """BASELINE.json configs[4] shapes: 256 experts, 8 bins, sigma ~ U[0.78,1.0]."""
    E, G, k = 256, 8, 8
    ids, _, counts = O.route_topk(I.make_logits(T, E, s, 3), E, k)
    load = counts.astype(np.float64)
    scale = I.make_throughput_scales(G, 3)
    bm, om = _models()[1]
    for cap in (0, E // G):
        a = B.placement_greedy(load, G, scale, bm, cap)
        assert np.array_equal(a, O.placement_greedy(load, G, scale, om, cap))
        tb = B.placement_token_balanced(load, G, cap)
        assert np.array_equal(tb, O.placement_token_balanced(load, G, cap))
        if cap:
            assert np.bincount(a, minlength=G).tolist() == [cap] * G
        for kind in (B.MODEL_A, B.MODEL_B):
            for asg in (a, tb, B.placement_contiguous(E, G)):
                assert B.placement_eval(asg, load, G, scale, bm, kind)[0] == pytest.approx(
                    O.placement_eval(asg, load, G, scale, om, kind)[0], rel=1e-12)
    assert np.array_equal(B.placement_contiguous(E, G), O.placement_contiguous(E, G))


def test_placement_invalid_arguments(lib):
    with pytest.raises(B.VibeError):
        B.placement_eval([0, 5], [1.0, 2.0], 2, [1.0, 1.0], None)
    with pytest.raises(B.VibeError):
        B.placement_greedy([1.0, 2.0, 3.0], 2, [1.0, 1.0], None, cap=1)
    with pytest.raises(B.VibeError):
        B.placement_greedy([1.0, 2.0], 2, [1.0, 0.0], None)
    with pytest.raises(B.VibeError):
        B.placement_eval([0, 1], [1.0, 2.0], 2, [1.0, 1.0], B.LatencyModel([2, 1], [1.0, 2.0], 1))


# ------------------------------------------------------------------ f1: recalibration (host code) vs oracle
def test_drift_cosine_and_monitor_match_oracle(lib):
    rng = I._rng(5, 5)
    for _ in range(20):
        a, b = rng.uniform(0, 50, 64), rng.uniform(0, 50, 64)
        assert B.drift_cosine(a, b) == O.cosine_distance(a, b)          # same operation order: bit-identical
    assert B.drift_cosine([0, 0], [1, 2]) == 0.0
    L, E = 3, 16
    bm, om = B.DriftMonitor(L, E, window=20, H=5, delta=0.05), O.DriftMonitor(L, E, window=20, H=5, delta=0.05)
    base = rng.uniform(1, 100, (L, E))
    shifted = base[:, ::-1].copy()
    ref_set = False
    for p in range(1, 161):
        mix = 0.0 if p < 60 else min(1.0, (p - 60) / 40.0)
        loads = np.floor((1 - mix) * base + mix * shifted + rng.uniform(0, 3, (L, E)))
        tb, db = bm.push(loads)
        to, do = om.push(loads)
        assert tb == to and (db is None) == (do is None)
        if db is not None:
            assert np.array_equal(db, do)
        if p == 20 and not ref_set:
            bm.set_reference(om.window_mean())
            om.set_reference(om.window_mean())
            assert np.array_equal(bm.window_mean(), om.window_mean())
            ref_set = True
        if tb:
            bm.rearranged()
            om.rearranged()
    assert om.passes == 160 and om.ref is not None
    bm.close()
    with pytest.raises(B.VibeError):
        B.DriftMonitor(0, 4)


def test_swap_refine_matches_oracle_and_golden(lib, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "swap_refine_worked_example.json")))
    a, swaps = B.placement_swap_refine(g["assign_start"], g["load"], 2, g["scale"], None, B.MODEL_A, g["eps"])
    assert a.tolist() == g["assign_final"] and [list(s) for s in swaps] == g["swaps"]
    n = g["no_reduction_case"]
    a, swaps = B.placement_swap_refine(n["assign_start"], n["load"], 2, n["scale"], None, B.MODEL_B, 0.03)
    assert a.tolist() == n["assign_start"] and swaps == []
    for (bm, om), kind, (E, G, seed) in itertools.product(_models(), (B.MODEL_A, B.MODEL_B),
                                                          [(16, 4, 0), (32, 8, 1), (64, 8, 2)]):
        rng = I._rng(seed, 78)
        load = np.floor(rng.pareto(1.2, E) * 40 + 1)
        scale = I.make_throughput_scales(G, seed)
        start = O.placement_contiguous(E, G)
        got, gs = B.placement_swap_refine(start, load, G, scale, bm, kind, 0.03)
        want, ws = O.placement_swap_refine(start, load, G, scale, om, kind, 0.03)
        assert np.array_equal(got, want) and gs == [tuple(map(int, s)) for s in ws]
        got1, gs1 = B.placement_swap_refine(start, load, G, scale, bm, kind, 0.03, max_swaps=2)
        assert gs1 == gs[:2]
    with pytest.raises(B.VibeError):
        B.placement_swap_refine([0, 3], [1.0, 2.0], 2, [1.0, 1.0], None)


def test_swap_refine_on_placement_stress_shape(lib):
    """configs[4] shape (256 experts, 8 bins, cap 32): a drifted load on a stale latency-balanced placement is
    repaired with few swaps (the paper reports 5-30 per layer versus > 200 moves for a full re-solve)."""
    E, G, k = 256, 8, 8
    bm, om = _models()[1]
    scale = I.make_throughput_scales(G, 3)
    old = O.route_topk(I.make_logits(16384, E, 1.2, 3), E, k)[2].astype(np.float64)
    new = O.route_topk(0.8 * I.make_logits(16384, E, 1.2, 3) + 0.2 * I.make_logits(16384, E, 1.2, 4), E, k)[2].astype(np.float64)
    stale = B.placement_greedy(old, G, scale, bm, E // G)
    before = B.placement_eval(stale, new, G, scale, bm, B.MODEL_B)[0]
    fixed, swaps = B.placement_swap_refine(stale, new, G, scale, bm, B.MODEL_B, 0.03)
    after, per = B.placement_eval(fixed, new, G, scale, bm, B.MODEL_B)
    assert after <= before and np.bincount(fixed, minlength=G).tolist() == [E // G] * G
    assert int((fixed != stale).sum()) <= 2 * len(swaps)          # every swap moves two experts
    resolve = B.placement_greedy(new, G, scale, bm, E // G)
    moved_full = int((resolve != stale).sum())
    assert 2 * len(swaps) <= moved_full or len(swaps) == 0
    want, ws = O.placement_swap_refine(stale, new, G, scale, om, O.MODEL_B, 0.03)
    assert np.array_equal(fixed, want)


def test_header_is_plain_c99(tmp_path):
    """include/vibe.h is the boundary: it must compile as C (no C++-isms, no torch types) and link against the library."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "t.c"
    src.write_text('#include "vibe.h"\n#include <stdio.h>\n'
                   'int main(void) { vibe_route_cfg c; (void)c;\n'
                   '  printf("%d %s %lld\\n", (int)vibe_version(), vibe_status_string(VIBE_ERR_WORKSPACE),\n'
                   '         (long long)vibe_rows_cap(64, 2, 8, 1)); return 0; }\n')
    exe = tmp_path / "t"
    build_mod.build()
    libdir = os.path.dirname(B.LIB_PATH)
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                        str(src), "-o", str(exe), "-L", libdir, "-lvibe", "-Wl,-rpath," + libdir],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.split() == ["100", "VIBE_ERR_WORKSPACE", "128"], (out.stdout, out.stderr)
