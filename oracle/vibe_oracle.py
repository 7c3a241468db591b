"""CPU ORACLE for the ViBE per-GPU MoE-layer hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  The product (paper_2606_00735_b200/) never does, and
this module imports nothing from the product except nothing at all: inputs arrive
as numpy arrays produced by paper_2606_00735_b200.inputs (the seeded generators).

What it is: a plain, slow, obviously-correct numpy (fp64 unless stated) statement
of what each C-ABI call computes, written from PAPER.md (ViBE, arxiv 2606.00735)
and, where the paper is silent (it treats the fused MoE kernel as a black box,
PAPER.md L176/L220/L420), from the readings listed in DESIGN.md ("Readings").
No blocking, no fusion, no reordering beyond the definitions.

Citations:  P:L<n> = /root/reference/PAPER.md line n;  R*/P*/F*/C*/M*/L* = DESIGN.md reading ids (D* = the f1 recalibration readings).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function below is pinned to
something other than itself -- brute force, closed forms, library routines
(scipy.special.softmax/expit, np.argsort(kind='stable'), torch CPU fp64 matmul+silu),
hand-worked golden fixtures in tests/golden/; the FP8 parts (O11, O12) additionally to torch's own
float8_e4m3fn / float8_e8m0fnu casts and to golden rows worked in exact rational arithmetic.
parity unpinned: only the latency *profile* (a measurement; nothing to pin numerically) -- its *model*
(O5) is pinned.
"""
from __future__ import annotations

import itertools
import numpy as np

SCORE_SOFTMAX = 0
SCORE_SIGMOID = 1

# ======================================================================================
# bf16 helpers (the oracle's own copy; the CUDA path has its own)
# ======================================================================================

def bf16_bits_to_f64(b):
    """bf16 bit pattern (uint16) -> exact value in f64."""
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16_bits(x):
    """Round an f64 array to bf16 with round-to-nearest-even, in one rounding
    (not via f32, which could double-round).  Inputs must be finite and within
    bf16 normal range or zero (true for every tensor on this path; F4)."""
    x = np.asarray(x, dtype=np.float64)
    m, e = np.frexp(x)                     # x = m * 2^e, 0.5 <= |m| < 1
    # bf16 has 8 significant bits: quantum = 2^(e-8); subnormal floor at 2^-133
    q = np.ldexp(1.0, np.maximum(e - 8, -133))
    r = np.rint(x / q) * q                 # np.rint = round-half-to-even
    r32 = r.astype(np.float32)             # exact: r has <= 8 significant bits
    u = r32.view(np.uint32)
    assert np.all((u & np.uint32(0xFFFF)) == 0), "bf16 rounding produced non-bf16 value"
    return (u >> np.uint32(16)).astype(np.uint16)


def bf16_round_f64(x):
    """x (f64) -> nearest bf16 value, returned as f64."""
    return bf16_bits_to_f64(f64_to_bf16_bits(x))


# ======================================================================================
# O1  route top-k  +  O1.6 activation histogram      (a1, a2)
# The paper only says "route each token to a subset of experts" and
# profiles "expert activation" into W in R^{LxE}.  Readings R1-R8.
# ======================================================================================

_F = np.float32
_LOG2E = _F(1.4426950408889634)
_LN2_HI = _F(0.693359375)            # 355/512, 9 significant bits: n*LN2_HI exact for |n|<2^15
_LN2_LO = _F(-2.12194440e-4)         # ln2 - LN2_HI
_VSIG_COEF = [_F(1.0 / 5040.0), _F(1.0 / 720.0), _F(1.0 / 120.0), _F(1.0 / 24.0),
              _F(1.0 / 6.0), _F(0.5), _F(1.0), _F(1.0)]      # Taylor e^r, degree 7, high -> low


def vsig_f32(x):
    """Reproducible f32 sigmoid used ONLY as the selection key (reading R2).

    Defined as this exact sequence of individually, correctly rounded IEEE-754
    binary32 operations (no fused multiply-add anywhere), so that a CPU and a GPU
    evaluating it agree bit for bit:
        x  = min(max(x,-80),80);  a = -x
        n  = rint(a*LOG2E)                       (round half to even)
        r  = (a - n*LN2_HI) - n*LN2_LO           (Cody-Waite; 3 roundings)
        p  = (((((((c7*r + c6)*r + c5)*r + c4)*r + c3)*r + c2)*r + c1)*r + c0
             each * and each + rounded separately; c_j = f32(1/j!)
        e  = p * 2^n                             (exact scaling; |n| <= 116 keeps it normal)
        vsig = 1 / (1 + e)                       (one add, one IEEE division)
    numpy evaluates every ufunc on float32 arrays as a separate correctly rounded
    binary32 operation, which is exactly this definition.
    """
    x = np.asarray(x, dtype=_F)
    x = np.minimum(np.maximum(x, _F(-80.0)), _F(80.0))
    a = -x
    n = np.rint(a * _LOG2E)
    r = a - n * _LN2_HI
    r = r - n * _LN2_LO
    p = np.full_like(r, _VSIG_COEF[0])
    for c in _VSIG_COEF[1:]:
        p = p * r
        p = p + c
    e = np.ldexp(p, n.astype(np.int32))
    assert e.dtype == _F
    one = _F(1.0)
    return one / (one + e)


def _argmax_untaken(v, taken):
    """Per row: the lowest index among the largest entries of v that are not `taken` (R3).  The k picks (and the
    topk_group kept groups) are k DISTINCT experts (groups) also when fewer than k entries are finite -- keys of
    -inf, e.g. masked logits or a group limit that leaves fewer than k finite keys: marking a pick by overwriting
    its key with -inf would then pick it again."""
    m = np.where(taken, -np.inf, v).max(axis=1, keepdims=True)
    return np.argmax((v == m) & ~taken, axis=1)              # first True = lowest index


def route_topk(logits, num_experts, top_k, score_fn=SCORE_SOFTMAX, renormalize=1,
               routed_scale=1.0, n_group=0, topk_group=0, select_bias=None):
    """O1 steps 1-6.  logits f32 [T,E] -> (topk_ids i32 [T,k], topk_w f32 [T,k], counts i32 [E]).

    1. x[e] = logits[t,e]
    2. key: softmax -> x (select on the raw logits, softmax is monotone; R2);
            sigmoid -> vsig(x) + select_bias (one f32 add; bias is selection-only; R1,R7)
    3. group limiting (R6): contiguous groups of E/n_group; group score = largest key +
       second largest key (one f32 add); keep the topk_group best groups (ties -> lower
       group index); key = -inf elsewhere
    4. k rounds of arg-max, ties -> lowest expert index (R3); ids in pick order
    5. weights in f64, rounded once to f32: softmax over ALL E experts (R1) or the true
       sigmoid 1/(1+e^-x) (bias excluded); optional renormalisation over the k picked
       (R4: no epsilon); times routed_scale (R5)
    6. counts[e] = number of assignments with id e, over GLOBAL experts (R8; one row of
       the activation matrix W of P:L178)
    """
    x = np.ascontiguousarray(logits, dtype=np.float32)
    T, E = x.shape
    k = int(top_k)
    assert E == num_experts and 1 <= k <= E
    # step 2
    if score_fn == SCORE_SOFTMAX:
        key = x.copy()
    else:
        s32 = vsig_f32(x)
        key = s32 if select_bias is None else (s32 + np.asarray(select_bias, dtype=_F)[None, :])
        assert key.dtype == _F
    key = key + _F(0.0)                      # -0.0 -> +0.0 (they compare equal anyway)
    # step 3
    if n_group and n_group > 1:
        assert E % n_group == 0 and 1 <= topk_group <= n_group and topk_group * (E // n_group) >= k
        gs = E // n_group
        kg = key.reshape(T, n_group, gs)
        srt = np.sort(kg, axis=2)
        if gs >= 2:
            gscore = srt[:, :, -1] + srt[:, :, -2]          # f32 add: larger + second
        else:
            gscore = srt[:, :, -1]
        assert gscore.dtype == _F
        keep = np.zeros((T, n_group), dtype=bool)
        for _ in range(topk_group):
            best = _argmax_untaken(gscore, keep)             # lowest group index among the best not yet kept
            keep[np.arange(T), best] = True
        key = np.where(np.repeat(keep, gs, axis=1), key, _F(-np.inf)).astype(_F)
    # step 4
    ids = np.empty((T, k), dtype=np.int32)
    taken = np.zeros((T, E), dtype=bool)
    rows = np.arange(T)
    for j in range(k):
        best = _argmax_untaken(key, taken)                   # lowest index among the largest keys not yet picked
        ids[:, j] = best
        taken[rows, best] = True
    # step 5
    xd = x.astype(np.float64)
    if score_fn == SCORE_SOFTMAX:
        ex = np.exp(xd - xd.max(axis=1, keepdims=True))
        p = ex / ex.sum(axis=1, keepdims=True)
    else:
        p = 1.0 / (1.0 + np.exp(-xd))
    w = np.take_along_axis(p, ids.astype(np.int64), axis=1)
    if renormalize:
        w = w / w.sum(axis=1, keepdims=True)
    w = w * float(routed_scale)
    # step 6
    counts = np.zeros(E, dtype=np.int32)
    for e in ids.ravel():
        counts[e] += 1
    return ids, w.astype(np.float32), counts


# ======================================================================================
# O2  permute  (a3): stable counting sort of assignments by local expert slot.
# "token dispatch remains local" on one GPU; readings P1-P4.
# ======================================================================================

def permute(X_bits, topk_ids, expert_map, E_loc, align=1):
    """X bf16 bits [T,d]; topk_ids [T,k]; expert_map[E] -> slot or -1 (None = identity).
    Returns offsets[E_loc+1], row_to_assign[R_cap], assign_to_row[A], Xp bits [R_cap,d], R
    where R_cap = offsets[E_loc] and R = number of real rows."""
    T, k = topk_ids.shape
    A = T * k
    flat = topk_ids.reshape(-1)
    E = int(flat.max()) + 1 if expert_map is None else len(expert_map)
    emap = np.arange(E, dtype=np.int32) if expert_map is None else np.asarray(expert_map, dtype=np.int32)
    cnt = np.zeros(E_loc, dtype=np.int64)
    for i in range(A):
        s = emap[flat[i]]
        if s >= 0:
            cnt[s] += 1
    offsets = np.zeros(E_loc + 1, dtype=np.int32)
    for s in range(E_loc):
        offsets[s + 1] = offsets[s] + ((cnt[s] + align - 1) // align) * align
    R_cap = int(offsets[E_loc])
    row_to_assign = np.full(R_cap, -1, dtype=np.int32)
    assign_to_row = np.full(A, -1, dtype=np.int32)
    Xp = np.zeros((R_cap, X_bits.shape[1]), dtype=np.uint16)
    fill = np.zeros(E_loc, dtype=np.int64)
    for i in range(A):                       # walk assignments in flat order => stable
        s = emap[flat[i]]
        if s < 0:
            continue
        r = int(offsets[s] + fill[s])
        fill[s] += 1
        row_to_assign[r] = i
        assign_to_row[i] = r
        Xp[r, :] = X_bits[i // k, :]
    return offsets, row_to_assign, assign_to_row, Xp, int(cnt.sum())


# ======================================================================================
# O3  grouped SwiGLU FFN (a4): the "fused MoE kernel" ViBE profiles;
# the dominant cost (49 % of prefill).  Readings F1-F4, C2.
# ======================================================================================

def swiglu_ffn_rows(x_bits, W1_bits, W3_bits, W2_bits, round_h=True, round_y=False):
    """One expert on a block of rows.  x bf16 bits [n,d]; W1,W3 [d,f]; W2 [f,d].
       g = x W1 ; u = x W3 ; h = bf16_rne( g/(1+exp(-g)) * u ) ; y = h W2     (all sums in f64)
    round_h: H is an MMA operand by contract (F2) -> rounded to bf16.
    round_y: additionally round Y to bf16 (the 'mirrored' reference; C2 uses round_y=False)."""
    x = bf16_bits_to_f64(x_bits)
    g = x @ bf16_bits_to_f64(W1_bits)
    u = x @ bf16_bits_to_f64(W3_bits)
    h = (g / (1.0 + np.exp(-g))) * u
    if round_h:
        h = bf16_round_f64(h)
    y = h @ bf16_bits_to_f64(W2_bits)
    if round_y:
        y = bf16_round_f64(y)
    return y, h


def grouped_ffn(Xp_bits, offsets, row_to_assign, W1_bits, W3_bits, W2_bits,
                round_h=True, round_y=False, rows=None):
    """Y f64 [R_cap,d] (and H f64 [R_cap,f]); padding rows (row_to_assign<0) stay zero.
    `rows`: optional iterable of row indices to compute (others left NaN) -- used for
    sampled parity at full size."""
    E_loc = len(offsets) - 1
    R_cap, d = Xp_bits.shape
    f = W1_bits.shape[2]
    Y = np.zeros((R_cap, d), dtype=np.float64)
    H = np.zeros((R_cap, f), dtype=np.float64)
    if rows is not None:
        Y[:] = np.nan
        H[:] = np.nan
        rows = np.asarray(sorted(set(int(r) for r in rows)), dtype=np.int64)
    for s in range(E_loc):
        lo, hi = int(offsets[s]), int(offsets[s + 1])
        sel = np.arange(lo, hi, dtype=np.int64)
        if rows is not None:
            sel = rows[(rows >= lo) & (rows < hi)]
        sel = sel[row_to_assign[sel] >= 0] if len(sel) else sel
        if len(sel) == 0:
            continue
        y, h = swiglu_ffn_rows(Xp_bits[sel], W1_bits[s], W3_bits[s], W2_bits[s], round_h, round_y)
        Y[sel] = y
        H[sel] = h
    if rows is not None:
        pad = np.nonzero(row_to_assign < 0)[0]
        Y[pad] = 0.0
        H[pad] = 0.0
    return Y, H


def ffn_naive_triple_loop(x_bits, W1_bits, W3_bits, W2_bits):
    """Pure-Python triple loops for tiny shapes (pin for swiglu_ffn_rows); math.fsum-free,
    plain left-to-right f64 accumulation."""
    import math
    x = bf16_bits_to_f64(x_bits).tolist()
    W1 = bf16_bits_to_f64(W1_bits).tolist()
    W3 = bf16_bits_to_f64(W3_bits).tolist()
    W2 = bf16_bits_to_f64(W2_bits).tolist()
    n, d, f = len(x), len(W1), len(W1[0])
    Y = [[0.0] * d for _ in range(n)]
    for r in range(n):
        h = [0.0] * f
        for j in range(f):
            g = 0.0
            u = 0.0
            for c in range(d):
                g += x[r][c] * W1[c][j]
                u += x[r][c] * W3[c][j]
            h[j] = (g / (1.0 + math.exp(-g))) * u
        hb = bf16_round_f64(np.array(h)).tolist()
        for m in range(d):
            acc = 0.0
            for j in range(f):
                acc += hb[j] * W2[j][m]
            Y[r][m] = acc
    return np.array(Y)


# ======================================================================================
# O4  weighted un-permute / combine (a5).  Reading C1.
# ======================================================================================

def combine(Y, assign_to_row, topk_w, T, k, round_out=False):
    """out[t,:] = sum_j (f64)w[t,j] * Y[assign_to_row[t*k+j],:] over resident j, slot order."""
    d = Y.shape[1]
    out = np.zeros((T, d), dtype=np.float64)
    w = np.asarray(topk_w, dtype=np.float32).astype(np.float64).reshape(T, k)
    a2r = np.asarray(assign_to_row).reshape(T, k)
    for t in range(T):
        for j in range(k):
            r = a2r[t, j]
            if r >= 0:
                out[t, :] += w[t, j] * Y[r, :]
    if round_out:
        out = bf16_round_f64(out)
    return out


def moe_layer_direct(X_bits, topk_ids, topk_w, expert_map, W1_bits, W3_bits, W2_bits, tokens=None,
                     return_abs=False):
    """Independent statement of the whole layer with NO permutation:
       out[t] = sum_j w[t,j] * FFN_{slot(id[t,j])}(x_t)   (non-resident experts contribute 0).
    Used to pin permute+ffn+combine together, and as the sampled full-size reference.
    return_abs: also return sum_j w[t,j]*|FFN(x_t)| per element, the quantity that bounds the
    error contributed by storing Y in bf16."""
    T, k = topk_ids.shape
    d = X_bits.shape[1]
    toks = range(T) if tokens is None else tokens
    out, out_abs = {}, {}
    for t in toks:
        acc = np.zeros(d, dtype=np.float64)
        acc_abs = np.zeros(d, dtype=np.float64)
        for j in range(k):
            s = topk_ids[t, j] if expert_map is None else expert_map[topk_ids[t, j]]
            if s < 0:
                continue
            y, _ = swiglu_ffn_rows(X_bits[t:t + 1], W1_bits[s], W3_bits[s], W2_bits[s])
            wj = float(np.float32(topk_w[t, j]))
            acc += wj * y[0]
            acc_abs += wj * np.abs(y[0])
        out[t] = acc
        out_abs[t] = acc_abs
    if tokens is None:
        out = np.stack([out[t] for t in range(T)])
        out_abs = np.stack([out_abs[t] for t in range(T)])
    return (out, out_abs) if return_abs else out


# ======================================================================================
# O5  latency model  f(n)  from profiled points  (a6 -> a7).  P:L176 "produces a function
# f_g(n) that maps token load n to expected kernel latency"; form unspecified -> M1.
# ======================================================================================

class LatencyModel:
    """Monotone piecewise-linear per-expert latency l(n) [us] with l(0)=0, linear
    extrapolation with the last segment's slope (M1).  E_prof = experts resident when
    profiled in uniform mode (M2), so the whole-kernel latency is F(n) = E_prof*l(n/E_prof)."""

    def __init__(self, tokens, latency_us, E_prof=1):
        t = np.asarray(tokens, dtype=np.float64)
        l = np.asarray(latency_us, dtype=np.float64)
        assert t.ndim == 1 and t.shape == l.shape and len(t) >= 1 and np.all(np.diff(t) > 0) and t[0] > 0
        self.tokens = np.concatenate([[0.0], t])
        self.lat = np.concatenate([[0.0], np.maximum.accumulate(l)])   # enforce non-decreasing
        self.E_prof = int(E_prof)

    def per_expert(self, n):
        n = float(n)
        t, l = self.tokens, self.lat
        if n <= 0.0:
            return 0.0
        if n >= t[-1]:
            slope = (l[-1] - l[-2]) / (t[-1] - t[-2])
            return float(l[-1] + slope * (n - t[-1]))
        i = int(np.searchsorted(t, n, side="right")) - 1
        return float(l[i] + (l[i + 1] - l[i]) * (n - t[i]) / (t[i + 1] - t[i]))

    def whole_kernel(self, n_total):
        return self.E_prof * self.per_expert(float(n_total) / self.E_prof)


# ======================================================================================
# O6  placement evaluator (a7):  T = max_g f_g(n_g),  n_g = sum_{e in S_g} w_e
# with f_g(n) = f(n)/sigma_g (M5).  model kind A: scalar f(n_g) (paper); kind B: per-expert sum (L4).
# ======================================================================================

MODEL_A = 0
MODEL_B = 1


def placement_eval(assign, load, G, scale, model, model_kind=MODEL_B):
    """Returns (score, per_bin[G])."""
    assign = np.asarray(assign)
    load = np.asarray(load, dtype=np.float64)
    per_bin = np.zeros(G, dtype=np.float64)
    for g in range(G):
        members = [e for e in range(len(load)) if assign[e] == g]
        if model_kind == MODEL_A:
            n_g = 0.0
            for e in members:
                n_g += load[e]
            L = model.whole_kernel(n_g)
        else:
            L = 0.0
            for e in members:
                L += model.per_expert(load[e])
        per_bin[g] = L / float(scale[g])
    return float(per_bin.max()), per_bin


# ======================================================================================
# O7  greedy placement (a8):  Algorithm 1 Phase 2 (prose P:L186-L196)
#     N = sum_e w_e ; s_g = 1/f_g(N/E) ; tau_g = N s_g / sum_h s_h ;
#     experts in descending w_e ; assign e to argmax_g (tau_g - n_g) ; n_g += w_e
# Readings L1 (cap), L2 (ties), L3 (token-balanced = sigma==1), M5/M6.
# ======================================================================================

def placement_greedy(load, G, scale, model, cap=0):
    load = np.asarray(load, dtype=np.float64)
    E = len(load)
    N = 0.0
    for e in range(E):
        N += load[e]
    n_ref = N / E
    fref = model.whole_kernel(n_ref) if model is not None else 1.0
    s = np.array([1.0 / (fref / float(scale[g])) if fref > 0 else float(scale[g]) for g in range(G)])
    ssum = 0.0
    for g in range(G):
        ssum += s[g]
    tau = np.array([N * s[g] / ssum for g in range(G)])
    order = sorted(range(E), key=lambda e: (-load[e], e))        # stable: ties -> lower e
    n = np.zeros(G, dtype=np.float64)
    cnt = np.zeros(G, dtype=np.int64)
    assign = np.full(E, -1, dtype=np.int32)
    for e in order:
        best, best_gap = -1, 0.0
        for g in range(G):
            if cap > 0 and cnt[g] >= cap:
                continue
            gap = tau[g] - n[g]
            if best < 0 or gap > best_gap:                      # strict > : ties -> lower g
                best, best_gap = g, gap
        assert best >= 0, "cap*G < E"
        assign[e] = best
        n[best] += load[e]
        cnt[best] += 1
    return assign


def placement_token_balanced(load, G, cap=0):
    """'EPLB implicitly assumes f_g(n)=n': the same greedy with all sigma equal."""
    return placement_greedy(load, G, np.ones(G), None, cap)


def placement_contiguous(E, G):
    """vLLM's default: expert e -> GPU floor(e*G/E)."""
    return np.array([(e * G) // E for e in range(E)], dtype=np.int32)


# ======================================================================================
# O8  brute force over all G^E labelled binnings (tests only; NP-hard in general)
# ======================================================================================

def placement_brute_force(load, G, scale, model, model_kind=MODEL_B, cap=0):
    E = len(load)
    best_score, best_assign = np.inf, None
    for a in itertools.product(range(G), repeat=E):
        if cap > 0 and max(a.count(g) for g in range(G)) > cap:
            continue
        sc, _ = placement_eval(a, load, G, scale, model, model_kind)
        if sc < best_score:
            best_score, best_assign = sc, np.array(a, dtype=np.int32)
    return best_score, best_assign


# ======================================================================================
# O9  drift detector (f1):  d = 1 - (w . w_ref) / (|w| |w_ref|)
#     "Every H forward passes (default H=10) ... cosine distance between the current
#     100-sample window average w and the reference ... When any layer's d exceeds a
#     threshold delta_cos (default 0.05) ... triggers the incremental solver";
#     Alg. 1 Phase 3: snapshot := current w at a rearrangement, then
#     "Cooldown for H forward passes".  Readings D1, D3.
# ======================================================================================

def cosine_distance(w, w_ref):
    w = np.asarray(w, dtype=np.float64)
    r = np.asarray(w_ref, dtype=np.float64)
    dot = 0.0
    nw = 0.0
    nr = 0.0
    for e in range(len(w)):
        dot += w[e] * r[e]
        nw += w[e] * w[e]
        nr += r[e] * r[e]
    if nw == 0.0 or nr == 0.0:
        return 0.0                                    # D1: a zero vector carries no direction
    return 1.0 - dot / (np.sqrt(nw) * np.sqrt(nr))


class DriftMonitor:
    """Alg. 1 Phase 3 bookkeeping for L layers x E experts (D3): a sliding window of the last
    `window` per-pass load vectors; every H-th pass, if a reference exists and no cooldown is
    running, d_l = cosine_distance(window mean_l, reference_l); trigger iff max_l d_l > delta."""

    def __init__(self, L, E, window=100, H=10, delta=0.05):
        self.L, self.E, self.window, self.H, self.delta = L, E, window, H, delta
        self.samples = []          # most recent `window` pushes, each [L,E]
        self.ref = None
        self.passes = 0
        self.cooldown = 0

    def window_mean(self):
        acc = np.zeros((self.L, self.E), dtype=np.float64)
        for s in self.samples:
            acc += s
        return acc / max(1, len(self.samples))

    def set_reference(self, W):
        self.ref = np.array(W, dtype=np.float64).reshape(self.L, self.E)

    def rearranged(self):
        """'w_ref <- w for all l; Cooldown for H forward passes'."""
        self.ref = self.window_mean()
        self.cooldown = self.H

    def push(self, loads):
        """One forward pass.  Returns (triggered, d[L] or None when no check ran)."""
        self.samples.append(np.array(loads, dtype=np.float64).reshape(self.L, self.E))
        if len(self.samples) > self.window:
            self.samples.pop(0)
        self.passes += 1
        if self.cooldown > 0:
            self.cooldown -= 1
            return False, None
        if self.ref is None or self.passes % self.H != 0:
            return False, None
        w = self.window_mean()
        d = np.array([cosine_distance(w[l], self.ref[l]) for l in range(self.L)])
        return bool(d.max() > self.delta), d


# ======================================================================================
# O10  incremental placement update (f1): Algorithm 2 (prose P:L210-L214, L426-L428)
#     repeat: g+ = slowest GPU, g- = fastest GPU; best swap (e_i in g+, e_j in g-) "maximizing
#     latency reduction"; swap; until max_g f_g(n_g) <= (1+eps) * mean_g f_g(n_g) "or no
#     latency reduction".  Reading D2: the reduction of a swap is max(L_g+, L_g-) before minus
#     after; ties -> lowest (e_i, e_j); argmax/argmin ties -> lower g.
# ======================================================================================

def bin_latencies(assign, load, G, scale, model, model_kind):
    return placement_eval(assign, load, G, scale, model, model_kind)[1]


def placement_swap_refine(assign, load, G, scale, model, model_kind=MODEL_B, eps=0.03, max_swaps=1 << 30):
    """Returns (assign', swaps) with swaps = [(e_i, e_j), ...] in the order applied."""
    assign = np.array(assign, dtype=np.int32)
    load = np.asarray(load, dtype=np.float64)
    swaps = []
    while len(swaps) < max_swaps:
        Lg = bin_latencies(assign, load, G, scale, model, model_kind)
        mean = 0.0
        for g in range(G):
            mean += Lg[g]
        mean /= G
        g_hi = int(np.argmax(Lg))          # first maximum: ties -> lower g
        g_lo = int(np.argmin(Lg))
        if Lg[g_hi] <= (1.0 + eps) * mean or g_hi == g_lo:
            break
        before = max(Lg[g_hi], Lg[g_lo])
        best, best_red = None, 0.0
        for ei in range(len(load)):
            if assign[ei] != g_hi:
                continue
            for ej in range(len(load)):
                if assign[ej] != g_lo:
                    continue
                trial = assign.copy()
                trial[ei], trial[ej] = g_lo, g_hi
                Lt = bin_latencies(trial, load, G, scale, model, model_kind)
                red = before - max(Lt[g_hi], Lt[g_lo])
                if red > best_red:                     # strict: ties -> first (lowest e_i, then e_j)
                    best, best_red = (ei, ej), red
        if best is None:
            break                                      # "no latency reduction"
        ei, ej = best
        assign[ei], assign[ej] = g_lo, g_hi
        swaps.append(best)
    return assign, swaps


# ======================================================================================
# O11  FP8 (e4m3) grouped FFN (f2).  The paper runs both models in FP8 (Table 2a) but says
#      nothing about the recipe; reading Q1-Q4: OCP e4m3 ("fn": no infinities, max 448,
#      round-to-nearest-even, saturating), per-expert weight scales absmax/448, per-row activation
#      scales rowabsmax/448, a STATIC per-expert scale for the intermediate H, products accumulated
#      exactly (f64 here, fp32 in the tensor core), scales applied to the accumulators.
# ======================================================================================

E4M3_MAX = 448.0


def e4m3_decode_table():
    """All 256 codes of OCP FP8 E4M3 (fn): 1 sign, 4 exponent (bias 7), 3 mantissa bits; exponent field 0 =
    subnormals (m/8 * 2^-6); S.1111.111 = NaN; no infinities."""
    t = np.zeros(256, dtype=np.float64)
    for code in range(256):
        sgn = -1.0 if code & 0x80 else 1.0
        ex = (code >> 3) & 0xF
        m = code & 0x7
        if ex == 0xF and m == 0x7:
            t[code] = np.nan
        elif ex == 0:
            t[code] = sgn * (m / 8.0) * 2.0 ** -6
        else:
            t[code] = sgn * (1.0 + m / 8.0) * 2.0 ** (ex - 7)
    return t


def e4m3_encode_scalar(x):
    """f64 -> e4m3 codes (uint8): round to nearest, ties to even mantissa, saturate at +-448 (no NaN made).
    The definition, element by element (slow); e4m3_encode below is the same arithmetic on whole arrays and
    is pinned against this one."""
    x = np.asarray(x, dtype=np.float64)
    out = np.zeros(x.shape, dtype=np.uint8)
    flat, o = x.reshape(-1), out.reshape(-1)
    for i in range(flat.size):
        v = flat[i]
        sgn = 0x80 if (v < 0 or (v == 0 and np.signbit(v))) else 0
        a = min(abs(v), E4M3_MAX)
        if a < 2.0 ** -6:                       # subnormal range: step 2^-9
            q = a / 2.0 ** -9
            n = int(np.floor(q))
            r = q - n
            if r > 0.5 or (r == 0.5 and (n & 1)):
                n += 1
            o[i] = sgn | n                      # n = 8 rolls over into the first normal (0001.000) correctly
            continue
        ex = int(np.floor(np.log2(a)))
        if 2.0 ** ex > a:                        # guard log2 rounding
            ex -= 1
        q = a / 2.0 ** ex * 8.0 - 8.0            # mantissa in [0, 8)
        n = int(np.floor(q))
        r = q - n
        if r > 0.5 or (r == 0.5 and (n & 1)):
            n += 1
        if n == 8:
            n, ex = 0, ex + 1
        code = ((ex + 7) << 3) | n
        o[i] = sgn | min(code, 0x7E)            # 0x7E = 448
    return out


def e4m3_encode(x):
    """The same rounding as e4m3_encode_scalar on whole arrays: |v| clamped to 448 = n * 2^(ex-3) with
    ex = max(floor(log2 |v|), -6) and n = rint(|v| / 2^(ex-3)) (np.rint: ties to even n, i.e. to the even
    mantissa); code = ((ex + 6) << 3) + n  (n < 8: subnormal; n = 16: carries into the next exponent)."""
    x = np.asarray(x, dtype=np.float64)
    a = np.minimum(np.abs(x), E4M3_MAX)
    _, fe = np.frexp(a)                          # a = m * 2^fe, 0.5 <= m < 1  ->  floor(log2 a) = fe - 1
    ex = np.maximum(fe - 1, -6)
    n = np.rint(a / np.ldexp(1.0, ex - 3)).astype(np.int64)
    code = ((ex.astype(np.int64) + 6) << 3) + n
    code = np.where(a == 0, 0, code)
    return (np.where(np.signbit(x), 0x80, 0) | code).astype(np.uint8)


def fp8_pack_weights(W_bits):
    """bf16 bits [E,K,N] -> (codes uint8 [E,N,K] (K contiguous), scale f32 [E] = absmax/448; all-zero expert: 1)."""
    W = bf16_bits_to_f64(W_bits)
    E = W.shape[0]
    scale = np.ones(E, dtype=np.float32)
    codes = np.zeros((E, W.shape[2], W.shape[1]), dtype=np.uint8)
    for e in range(E):
        amax = float(np.max(np.abs(W[e])))
        if amax > 0:
            scale[e] = np.float32(amax / E4M3_MAX)
        # Q3: the quantiser is an elementwise binary32 program (bf16 input widened to binary32, binary32 scale):
        # the quotient is the correctly rounded binary32 quotient, then rounded ONCE to e4m3.  Pinned by
        # tests/golden/fp8_quotient_precision_example.json (a row where the f64 quotient gives another code)
        codes[e] = e4m3_encode((W[e].T.astype(np.float32) / scale[e]).astype(np.float64))
    return codes, scale


def fp8_quantize_rows(X_bits):
    """bf16 bits [R,d] -> (codes uint8 [R,d], row_scale f32 [R] = rowabsmax/448; all-zero row: 1)."""
    X = bf16_bits_to_f64(X_bits)
    R = X.shape[0]
    scale = np.ones(R, dtype=np.float32)
    for r in range(R):
        amax = float(np.max(np.abs(X[r]))) if X.shape[1] else 0.0
        if amax > 0:
            scale[r] = np.float32(amax / E4M3_MAX)
    codes = (e4m3_encode((X.astype(np.float32) / scale[:, None]).astype(np.float64)) if R
             else np.zeros_like(X_bits, dtype=np.uint8))
    return codes, scale


def fp8_quantize_static(v, scale):
    """Q3 with a given scale: v -> binary32, quotient by the binary32 scale formed in binary32, ONE rounding to e4m3."""
    return e4m3_encode((np.asarray(v).astype(np.float32) / np.float32(scale)).astype(np.float64))


def grouped_ffn_fp8(Xq, row_scale, offsets, row_to_assign, W1q, s1, W3q, s3, W2q, s2, h_scale, Hq_given=None):
    """Per resident expert e and real row r:  g = sx[r] s1[e] (xq . w1q),  u = sx[r] s3[e] (xq . w3q),
    h = silu(g) u,  hq = e4m3(h / sh[e]),  y = sh[e] s2[e] (hq . w2q).  Returns (Y f64 [R,d], Hq codes [R,f]).
    Hq_given (codes [R,f]): the down projection runs on THESE codes instead of the ones computed here (the returned
    Hq is still the computed one) -- lets a parity test separate the two GEMMs: a code that the device decided one
    e4m3 step away (its h is an fp32 sum in an order no oracle can know) moves y by up to 2^-3 |h| |w2|."""
    T8 = e4m3_decode_table()
    R = int(offsets[-1])
    f, d = W1q.shape[1], W1q.shape[2]
    Y = np.zeros((R, d), dtype=np.float64)
    Hq = np.zeros((R, f), dtype=np.uint8)
    for e in range(len(offsets) - 1):
        lo, hi = int(offsets[e]), int(offsets[e + 1])
        rows = [r for r in range(lo, hi) if row_to_assign[r] >= 0]
        if not rows:
            continue
        x = T8[Xq[rows]]                                            # [n,d] exact e4m3 values
        sx = row_scale[rows].astype(np.float64)[:, None]
        g = (x @ T8[W1q[e]].T) * sx * np.float64(s1[e])
        u = (x @ T8[W3q[e]].T) * sx * np.float64(s3[e])
        h = g / (1.0 + np.exp(-g)) * u
        # Q3 applies to H as to X: the value is a binary32 number (the epilogue's), the quotient h/sh is formed
        # in binary32 and rounded ONCE to e4m3
        hq = fp8_quantize_static(h, h_scale[e])
        Hq[rows] = hq
        if Hq_given is not None:
            hq = np.asarray(Hq_given)[rows]
        Y[rows] = (T8[hq] @ T8[W2q[e]].T) * np.float64(h_scale[e]) * np.float64(s2[e])
    return Y, Hq


# ======================================================================================
# O12  Block-scaled FP8 ("MXFP8": e4m3 elements, one power-of-two UE8M0 scale per block of the contraction
#      dimension) grouped FFN (f2 as S8(f) words it: "e4m3, block-scaled").  The paper says only "Precision:
#      FP8" (Table 2a); readings Q5-Q8:
#      Q5  a block = `block` consecutive elements along K of one row (activations: a token row; weights: one
#          output feature), block = 32 (the OCP-MX / tensor-core native block) or 128 (DeepSeek-V3's
#          activation tile, stored as the same scale repeated over its four 32-blocks); scale = 2^e, stored
#          as the byte e + 127 (UE8M0), one byte per 32 elements in either case.
#      Q6  e = the smallest integer with amax <= 448 * 2^e (no element saturates), clamped to [-127, 127];
#          an all-zero block: e = 0.  x / 2^e is EXACT in binary arithmetic, so no quotient-precision
#          question arises (contrast Q3); one rounding, to e4m3 (RNE).
#      Q7  the intermediate H is block-scaled the same way, per row and 32 features, from its binary32 value.
#      Q8  products of the dequantised values (code value * 2^e, exact) accumulated in f64 (fp32 in the
#          tensor core); SwiGLU in f64; Y not rounded here (the caller rounds / compares, C2).
# ======================================================================================

MX_BLOCK = 32            # elements per stored scale byte


def ue8m0_exponent(amax):
    """Q6: smallest integer e with amax <= 448 * 2^e, clamped to [-127, 127]; amax == 0 -> 0.
    amax = m * 2^x with 1 <= m < 2:  448 = 1.75 * 2^8, so e = x - 8 if m <= 1.75 else x - 7."""
    amax = np.asarray(amax, dtype=np.float64)
    mant, ex = np.frexp(amax)                 # amax = mant * 2^ex, 0.5 <= mant < 1  ->  m = 2 mant, x = ex - 1
    e = np.where(mant <= 0.875, ex - 1 - 8, ex - 1 - 7)
    e = np.clip(e, -127, 127)
    return np.where(amax == 0, 0, e).astype(np.int64)


def mx_quantize(V, block=32):
    """V f64 [..., K] (K a multiple of `block`, block in {32, 128}) -> (codes uint8 [..., K],
    sf uint8 [..., K/32] = e + 127).  Block by block: amax, exponent (Q6), exact division, e4m3 RNE."""
    assert block in (32, 128)
    V = np.asarray(V, dtype=np.float64)
    K = V.shape[-1]
    assert K % block == 0
    lead = V.shape[:-1]
    Vb = V.reshape(lead + (K // block, block))
    e = ue8m0_exponent(np.max(np.abs(Vb), axis=-1))                      # [..., K/block]
    q = Vb / np.ldexp(1.0, e)[..., None]                                 # exact
    codes = e4m3_encode(q).reshape(V.shape)
    sf = np.repeat((e + 127).astype(np.uint8), block // MX_BLOCK, axis=-1)
    return codes, sf


def mx_dequantize(codes, sf):
    """codes [..., K], sf [..., K/32] -> exact f64 values code_value * 2^(sf - 127)."""
    T8 = e4m3_decode_table()
    return T8[codes] * np.repeat(np.ldexp(1.0, sf.astype(np.int64) - 127), MX_BLOCK, axis=-1)


def mx_pack_weights(W_bits, block=32):
    """bf16 bits [E,K,N] -> (codes uint8 [E,N,K] (K contiguous), sf uint8 [E,N,K/32]): one scale per
    output feature and K-block (Q5)."""
    W = bf16_bits_to_f64(W_bits)
    return mx_quantize(np.transpose(W, (0, 2, 1)), block)


def mx_quantize_rows(X_bits, block=32):
    """bf16 bits [R,d] -> (codes uint8 [R,d], sf uint8 [R,d/32])."""
    return mx_quantize(bf16_bits_to_f64(X_bits), block)


def grouped_ffn_mxfp8(Xq, Xsf, offsets, row_to_assign, W1q, W1sf, W3q, W3sf, W2q, W2sf, H_given=None):
    """Per resident expert e and real row r (Q8):  g = x . w1,  u = x . w3  on the dequantised values,
    h = silu(g) u,  (hq, hsf) = block-32 quantisation of binary32(h) along f (Q7),  y = deq(hq) . w2.
    Returns (Y f64 [R,d], Hq codes [R,f], Hsf [R,f/32]).
    H_given = (codes [R,f], scale bytes [R,f/32]): the down projection runs on THESE instead of the ones computed
    here (the returned Hq / Hsf are still the computed ones) -- separates the two GEMMs in a parity test, as in
    grouped_ffn_fp8."""
    R = int(offsets[-1])
    f, d = W1q.shape[1], W1q.shape[2]
    Y = np.zeros((R, d), dtype=np.float64)
    Hq = np.zeros((R, f), dtype=np.uint8)
    Hsf = np.full((R, f // MX_BLOCK), 127, dtype=np.uint8)
    for e in range(len(offsets) - 1):
        lo, hi = int(offsets[e]), int(offsets[e + 1])
        rows = [r for r in range(lo, hi) if row_to_assign[r] >= 0]
        if not rows:
            continue
        x = mx_dequantize(Xq[rows], Xsf[rows])                          # [n,d]
        g = x @ mx_dequantize(W1q[e], W1sf[e]).T
        u = x @ mx_dequantize(W3q[e], W3sf[e]).T
        h = g / (1.0 + np.exp(-g)) * u
        hq, hsf = mx_quantize(h.astype(np.float32).astype(np.float64), 32)
        Hq[rows], Hsf[rows] = hq, hsf
        if H_given is not None:
            hq, hsf = np.asarray(H_given[0])[rows], np.asarray(H_given[1])[rows]
        Y[rows] = mx_dequantize(hq, hsf) @ mx_dequantize(W2q[e], W2sf[e]).T
    return Y, Hq, Hsf


# ======================================================================================
# parity metrics (F3): max|err| / RMS(ref)  and  mean|err| / mean|ref|
# ======================================================================================

def ffn_error_metrics(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    err = np.abs(got - ref)
    rms = float(np.sqrt(np.mean(ref * ref)))
    mean_abs_ref = float(np.mean(np.abs(ref)))
    return {
        "max_abs_err_over_rms": float(err.max() / rms) if rms > 0 else float(err.max()),
        "mean_rel_err": float(err.mean() / mean_abs_ref) if mean_abs_ref > 0 else float(err.mean()),
        "rms_ref": rms,
    }
