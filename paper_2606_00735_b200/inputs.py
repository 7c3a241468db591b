"""Seeded synthetic inputs for the MoE-layer hot path (numpy only).

This module is the ONE piece shared by the CUDA path's tests/bench and by the
CPU oracle.  It holds no arithmetic of the method itself (no routing, no
permutation, no FFN, no combine, no placement): it only draws random arrays
with the shapes / value distributions / skew that BASELINE.json `configs`
prescribe and hands the identical arrays to both sides.

Recipe:
  * logits[T,E]  f32 = N(0,1) + alpha * zipf_bias(E, s)        (workload skew)
  * zipf_bias    : rank = permutation(E)+1 ; p ~ rank^-s ; bias = ln p - mean ln p
  * X[T,d]       bf16(RNE) of N(0,1)
  * W1,W3[E_loc,d,f] bf16 of N(0, 1/sqrt(d)); W2[E_loc,f,d] bf16 of N(0, 1/sqrt(f))
  * select_bias[E] f32 = N(0, 0.02^2)    (sigmoid configs only; selection-only bias)
bf16 tensors are carried as raw uint16 bit patterns so that both sides see the
same bits.  These synthetic tensors stand in for the ShareGPT / Sonnet traffic
and the DeepSeek-V3 / Qwen-3 / Mixtral weights used by the paper
(Tables 2a/2b), none of which exist in this container.
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np

SCORE_SOFTMAX = 0
SCORE_SIGMOID = 1


@dataclasses.dataclass(frozen=True)
class LayerConfig:
    """Shape + routing recipe of one MoE layer (BASELINE.json configs[i])."""
    name: str
    T: int            # tokens
    d: int            # hidden
    f: int            # expert intermediate
    E: int            # global experts
    k: int            # top-k
    E_loc: int        # resident experts (== E unless EP shard)
    score_fn: int = SCORE_SOFTMAX
    renormalize: int = 1
    routed_scale: float = 1.0
    n_group: int = 0
    topk_group: int = 0
    zipf_s: float = 0.0
    alpha: float = 1.0
    has_select_bias: bool = False

    @property
    def A(self) -> int:
        return self.T * self.k


# BASELINE.json configs[0..3]  (configs[4] is host-side placement; see placement tests)
C0 = LayerConfig("C0-tiny", T=64, d=256, f=512, E=8, k=2, E_loc=8, zipf_s=1.2)
C1 = LayerConfig("C1-mixtral-8x7b", T=4096, d=4096, f=14336, E=8, k=2, E_loc=8, zipf_s=0.5)
C2 = LayerConfig("C2-qwen3-30b-a3b", T=8192, d=2048, f=768, E=128, k=8, E_loc=128, zipf_s=1.0)
C3 = LayerConfig("C3-deepseek-v3-ep32", T=16384, d=7168, f=2048, E=256, k=8, E_loc=32,
                 score_fn=SCORE_SIGMOID, n_group=8, topk_group=4, zipf_s=1.2,
                 has_select_bias=True)
CONFIGS = {"C0": C0, "C1": C1, "C2": C2, "C3": C3}


def scaled(cfg: LayerConfig, **kw) -> LayerConfig:
    """A copy of cfg with some fields replaced (used for reduced-size parity cases)."""
    return dataclasses.replace(cfg, **kw)


# ----------------------------------------------------------------------------------
# bf16 as raw bits (data generation only: rounding a drawn f32 sample to bf16)
# ----------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even f32 -> bf16, returned as uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = u + np.uint32(0x7FFF) + lsb
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


# ----------------------------------------------------------------------------------
# generators
# ----------------------------------------------------------------------------------
def _rng(seed: int, *tags: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([int(seed), *[int(t) for t in tags]]))


def zipf_bias(E: int, s: float, seed: int, alpha: float = 1.0) -> np.ndarray:
    """Per-expert additive logit bias from Zipf(s) ranks (f32, zero-mean)."""
    if s == 0.0:
        return np.zeros(E, dtype=np.float32)
    rng = _rng(seed, 101)
    rank = rng.permutation(E).astype(np.float64) + 1.0
    lnp = -float(s) * np.log(rank)
    lnp = lnp - np.log(np.sum(np.exp(lnp)))
    return (alpha * (lnp - lnp.mean())).astype(np.float32)


def make_logits(T: int, E: int, s: float, seed: int, alpha: float = 1.0) -> np.ndarray:
    rng = _rng(seed, 102)
    z = rng.standard_normal((T, E), dtype=np.float32)
    z += zipf_bias(E, s, seed, alpha)[None, :]
    return z


def make_select_bias(E: int, seed: int) -> np.ndarray:
    return (_rng(seed, 103).standard_normal(E) * 0.02).astype(np.float32)


def make_X(T: int, d: int, seed: int) -> np.ndarray:
    return f32_to_bf16_bits(_rng(seed, 104).standard_normal((T, d), dtype=np.float32))


def make_expert_weight(which: int, e: int, rows: int, cols: int, std: float, seed: int) -> np.ndarray:
    """One expert's [rows, cols] weight matrix as bf16 bits. which: 1=W1(gate) 2=W2(down) 3=W3(up)."""
    w = _rng(seed, 200 + which, e).standard_normal((rows, cols), dtype=np.float32)
    w *= np.float32(std)
    return f32_to_bf16_bits(w)


def make_weights(E_loc: int, d: int, f: int, seed: int, out=None, threads: int | None = None):
    """W1,W3 [E_loc,d,f] and W2 [E_loc,f,d] as uint16 bf16 bits.  `out` may hold
    three preallocated uint16 arrays (e.g. views of pinned host tensors)."""
    if out is None:
        W1 = np.empty((E_loc, d, f), np.uint16)
        W3 = np.empty((E_loc, d, f), np.uint16)
        W2 = np.empty((E_loc, f, d), np.uint16)
    else:
        W1, W3, W2 = out
    std13 = 1.0 / np.sqrt(d)
    std2 = 1.0 / np.sqrt(f)

    def job(args):
        which, e = args
        if which == 1:
            W1[e] = make_expert_weight(1, e, d, f, std13, seed)
        elif which == 3:
            W3[e] = make_expert_weight(3, e, d, f, std13, seed)
        else:
            W2[e] = make_expert_weight(2, e, f, d, std2, seed)

    jobs = [(w, e) for e in range(E_loc) for w in (1, 3, 2)]
    nthr = threads or min(len(jobs), len(os.sched_getaffinity(0)))
    if nthr <= 1:
        for j in jobs:
            job(j)
    else:
        with ThreadPoolExecutor(nthr) as ex:
            list(ex.map(job, jobs))
    return W1, W3, W2


def make_expert_map(cfg: LayerConfig, policy: str = "contiguous", seed: int = 0) -> np.ndarray:
    """expert_map[E] -> local slot or -1.  'contiguous' = experts 0..E_loc-1 resident
    (vLLM's default placement); 'strided' = every (E/E_loc)-th expert;
    'random' = a seeded subset in shuffled slot order."""
    m = np.full(cfg.E, -1, dtype=np.int32)
    if policy == "contiguous":
        m[: cfg.E_loc] = np.arange(cfg.E_loc, dtype=np.int32)
    elif policy == "strided":
        step = cfg.E // cfg.E_loc
        m[::step][: cfg.E_loc] = np.arange(cfg.E_loc, dtype=np.int32)
    elif policy == "random":
        rng = _rng(seed, 105)
        chosen = rng.permutation(cfg.E)[: cfg.E_loc]
        m[chosen] = np.arange(cfg.E_loc, dtype=np.int32)
    else:
        raise ValueError(policy)
    return m


def make_layer(cfg: LayerConfig, seed: int = 0, with_weights: bool = True, map_policy: str = "contiguous"):
    """All inputs of one MoE layer as a dict of numpy arrays."""
    out = {
        "cfg": cfg,
        "logits": make_logits(cfg.T, cfg.E, cfg.zipf_s, seed, cfg.alpha),
        "select_bias": make_select_bias(cfg.E, seed) if cfg.has_select_bias else None,
        "X": make_X(cfg.T, cfg.d, seed),
        "expert_map": make_expert_map(cfg, map_policy, seed),
    }
    if with_weights:
        out["W1"], out["W3"], out["W2"] = make_weights(cfg.E_loc, cfg.d, cfg.f, seed)
    return out


def route_kwargs(cfg: LayerConfig) -> dict:
    return dict(num_experts=cfg.E, top_k=cfg.k, score_fn=cfg.score_fn, renormalize=cfg.renormalize,
                routed_scale=cfg.routed_scale, n_group=cfg.n_group, topk_group=cfg.topk_group)


# ----------------------------------------------------------------------------------
# placement-stress inputs (BASELINE.json configs[4])
# ----------------------------------------------------------------------------------
def make_throughput_scales(G: int, seed: int, lo: float = 0.78, hi: float = 1.0) -> np.ndarray:
    """sigma_g ~ U[lo,hi]: stand-in for the device-to-device DVFS/power/thermal spread
    (22 % in prior work)."""
    return _rng(seed, 106).uniform(lo, hi, size=G).astype(np.float64)


def balanced_ids(T: int, E: int, k: int, seed: int = 0) -> np.ndarray:
    """Perfectly balanced routing ids [T,k] (each expert gets T*k/E assignments, distinct
    experts per token): the 'perfect token balance' protocol of PAPER.md L108/L335."""
    assert (T * k) % E == 0 and k <= E
    t = np.arange(T, dtype=np.int64)[:, None]
    j = np.arange(k, dtype=np.int64)[None, :]
    return ((t * k + j) % E).astype(np.int32)
