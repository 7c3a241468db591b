// route.cu -- a1 + a2: top-k routing with fused expert-activation histogram (vibe_route_topk).
//
// One token per group of LANES lanes (LANES = 8 for small E, else a full warp); every lane
// keeps VPL consecutive experts' keys in registers (vectorised, coalesced 16-byte loads).
// Selection is k rounds of {local max, redux.sync max over the group, ballot, lowest lane
// wins} on order-preserving u32 images of the f32 keys, which gives the "ties -> lowest
// expert index" rule for free (lane-major element order).  The histogram is privatised in
// shared memory per block and merged with one global atomic per non-empty bin.
// Gate weights are evaluated in fp64 for the k picked experts only.
// Three kernels: route_topk_kernel (any E <= 512, k <= 32, any grouping), route_topk8_kernel (E = 128 | 256, k <= 8,
// four tokens per warp, (key, index) pairs: left with the un-renormalised softmax) and route_topk8p_kernel (the same
// shapes with no groups or 8 groups, sigmoid or renormalised softmax: packed one-register keys, merge networks, staged
// logits, approximate sigmoid keys with an exact redo where a margin fails -- the kernel of the C2 / C3 / 64K configs).
// The counts are zeroed by a one-block kernel that the route kernel overlaps (programmatic dependent launch).
//
// Semantics: include/vibe.h (vibe_route_topk), readings R1-R8.
#include <mutex>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

// counts <- 0.  The route kernels are launched with programmatic stream serialisation behind it: they start while it
// runs (everything older in the stream is complete: it is an ordinary launch) and wait for it (griddepcontrol.wait)
// only before they add their block histograms to the counts, so the zeroing costs no dependent launch latency.
__global__ void route_zero_counts_kernel(int32_t* counts, int E) {
  for (int i = threadIdx.x; i < E; i += blockDim.x) counts[i] = 0;
}

struct RouteParams {
  const float* logits;
  const float* bias;
  int32_t* ids;
  float* w;
  int32_t* counts;
  int T, E, k;
  int renorm;
  float scale;
  int n_group, topk_group;
  int fast_groups;  // 1: a lane's VPL experts lie in one group and lanes/group is a power of two
};

// ---- reproducible f32 sigmoid for the selection key (R2) ----------------------
// Exactly this sequence of separately rounded binary32 operations; no FMA contraction
// (explicit _rn intrinsics).  Constants are given by bit pattern.
__device__ __forceinline__ float vsig(float x) {
  const float LOG2E = __uint_as_float(0x3fb8aa3bu);   // 1.44269502
  const float LN2_HI = __uint_as_float(0x3f318000u);  // 0.693359375
  const float LN2_LO = __uint_as_float(0xb95e8083u);  // -2.12194442e-4
  x = fminf(fmaxf(x, -80.0f), 80.0f);
  const float a = -x;
  const float n = rintf(__fmul_rn(a, LOG2E));
  float r = __fsub_rn(a, __fmul_rn(n, LN2_HI));
  r = __fsub_rn(r, __fmul_rn(n, LN2_LO));
  float p = __uint_as_float(0x39500d01u);                               // 1/5040
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3ab60b61u));        // 1/720
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3c088889u));        // 1/120
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3d2aaaabu));        // 1/24
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3e2aaaabu));        // 1/6
  p = __fadd_rn(__fmul_rn(p, r), 0.5f);
  p = __fadd_rn(__fmul_rn(p, r), 1.0f);
  p = __fadd_rn(__fmul_rn(p, r), 1.0f);
  // exact scaling by 2^n: p in (0.70, 1.42) and |n| <= 116 keep the result normal
  const float e = __int_as_float(__float_as_int(p) + (__float2int_rn(n) << 23));
  return __fdiv_rn(1.0f, __fadd_rn(1.0f, e));
}

// order-preserving map f32 -> u32 (after -0 -> +0 so that -0 == +0 as in a float compare)
__device__ __forceinline__ uint32_t ordered_u32(float x) {
  const uint32_t b = __float_as_uint(__fadd_rn(x, 0.0f));
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

template <int LANES>
__device__ __forceinline__ uint32_t group_max_u32(unsigned gmask, uint32_t v) {
  return __reduce_max_sync(gmask, v);
}
template <int LANES>
__device__ __forceinline__ double group_sum_f64(unsigned gmask, double v) {
#pragma unroll
  for (int o = LANES / 2; o >= 1; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
  return v;
}

constexpr uint32_t kTaken = 0u;  // below ordered_u32(-inf) = 0x007fffff

template <int LANES, int VPL, bool SIGMOID>
__global__ void __launch_bounds__(256) route_topk_kernel(const RouteParams p) {
  extern __shared__ int s_mem[];
  int* s_hist = s_mem;                                        // [E]
  float* s_gscore = reinterpret_cast<float*>(s_mem + p.E);    // [groups_per_block][n_group] (generic path)
  for (int i = threadIdx.x; i < p.E; i += blockDim.x) s_hist[i] = 0;
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const int sub = lane % LANES;
  const unsigned gmask = (LANES == 32) ? 0xffffffffu : (((1u << LANES) - 1u) << (lane - sub));
  constexpr int kGroupsPerBlock = 256 / LANES;
  const int gidx = threadIdx.x / LANES;
  const int e0 = sub * VPL;
  const int E = p.E, k = p.k;
  const float NEG_INF = __int_as_float(0xff800000);
  const bool vec_ok = (VPL % 4 == 0) && (E % 4 == 0);

  float bias[VPL];
#pragma unroll
  for (int v = 0; v < VPL; ++v) bias[v] = (SIGMOID && p.bias != nullptr && e0 + v < E) ? p.bias[e0 + v] : 0.0f;

  for (int t = blockIdx.x * kGroupsPerBlock + gidx; t < p.T; t += gridDim.x * kGroupsPerBlock) {
    // ---- load this lane's VPL logits ----
    float x[VPL];
    const float* row = p.logits + (size_t)t * E;
    if (vec_ok) {
#pragma unroll
      for (int q = 0; q < VPL / 4; ++q) {
        if (e0 + 4 * q < E) {
          const uint4 u = ld_nc_v4(row + e0 + 4 * q);
          x[4 * q + 0] = __uint_as_float(u.x);
          x[4 * q + 1] = __uint_as_float(u.y);
          x[4 * q + 2] = __uint_as_float(u.z);
          x[4 * q + 3] = __uint_as_float(u.w);
        } else {
          x[4 * q + 0] = x[4 * q + 1] = x[4 * q + 2] = x[4 * q + 3] = NEG_INF;
        }
      }
    } else {
#pragma unroll
      for (int v = 0; v < VPL; ++v) x[v] = (e0 + v < E) ? __ldg(row + e0 + v) : NEG_INF;
    }
    // ---- selection keys ----
    float key[VPL];
    uint32_t uk[VPL];
#pragma unroll
    for (int v = 0; v < VPL; ++v) {
      if (SIGMOID) {
        key[v] = (e0 + v < E) ? __fadd_rn(vsig(x[v]), bias[v]) : NEG_INF;
      } else {
        key[v] = x[v];
      }
      uk[v] = ordered_u32(key[v]);
    }
    // ---- group-limited routing (R6) ----
    if (p.n_group > 1) {
      const int gs = E / p.n_group;
      if (p.fast_groups) {
        const int lpg = gs / VPL;  // lanes per group (power of two)
        float m1 = NEG_INF, m2 = NEG_INF;
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          const float c = key[v];
          if (c > m1) { m2 = m1; m1 = c; } else if (c > m2) { m2 = c; }
        }
        for (int o = 1; o < lpg; o <<= 1) {
          const float q1 = __shfl_xor_sync(gmask, m1, o);
          const float q2 = __shfl_xor_sync(gmask, m2, o);
          const float lo = fminf(m1, q1);
          m1 = fmaxf(m1, q1);
          m2 = fmaxf(lo, fmaxf(m2, q2));
        }
        const int g = e0 / gs;
        float score = (gs >= 2) ? __fadd_rn(m1, m2) : m1;
        if (e0 >= E) score = NEG_INF;
        int rank = 0;
        for (int g2 = 0; g2 < p.n_group; ++g2) {
          const float s2 = __shfl_sync(gmask, score, (lane - sub) + g2 * lpg);
          rank += (s2 > score || (s2 == score && g2 < g)) ? 1 : 0;
        }
        if (rank >= p.topk_group || e0 >= E) {
#pragma unroll
          for (int v = 0; v < VPL; ++v) uk[v] = ordered_u32(NEG_INF);
        }
      } else {
        // generic: one pass per group, scores parked in shared memory
        float* gsc = s_gscore + gidx * p.n_group;
        for (int g2 = 0; g2 < p.n_group; ++g2) {
          float m1 = NEG_INF, m2 = NEG_INF;
#pragma unroll
          for (int v = 0; v < VPL; ++v) {
            const int e = e0 + v;
            const float c = (e < E && e / gs == g2) ? key[v] : NEG_INF;
            if (c > m1) { m2 = m1; m1 = c; } else if (c > m2) { m2 = c; }
          }
#pragma unroll
          for (int o = 1; o < LANES; o <<= 1) {
            const float q1 = __shfl_xor_sync(gmask, m1, o);
            const float q2 = __shfl_xor_sync(gmask, m2, o);
            const float lo = fminf(m1, q1);
            m1 = fmaxf(m1, q1);
            m2 = fmaxf(lo, fmaxf(m2, q2));
          }
          if (sub == 0) gsc[g2] = (gs >= 2) ? __fadd_rn(m1, m2) : m1;
        }
        __syncwarp(gmask);
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          const int e = e0 + v;
          if (e < E) {
            const int g = e / gs;
            const float score = gsc[g];
            int rank = 0;
            for (int g2 = 0; g2 < p.n_group; ++g2) {
              const float s2 = gsc[g2];
              rank += (s2 > score || (s2 == score && g2 < g)) ? 1 : 0;
            }
            if (rank >= p.topk_group) uk[v] = ordered_u32(NEG_INF);
          }
        }
        __syncwarp(gmask);
      }
    }
    // ---- k rounds of arg-max, ties -> lowest index (R3) ----
    // Pick order = (key descending, expert index ascending).  Every lane keeps the FIRST TWO of its
    // not-yet-picked experts in that order (m1/v1, m2/v2) and the last one it gave away (lk/lv); a
    // round is then redux-max over the lane heads + ballot (lowest lane = lowest index among equal
    // keys) + a pop in the winner -- no scan of the VPL registers.  A lane that has given away both
    // of its candidates rebuilds them from its registers ("strictly after (lk, lv) in pick order");
    // with VPL experts per lane that happens about once per token.
    uint32_t lk = 0xffffffffu, m1 = kTaken, m2 = kTaken;
    int lv = -1, v1 = 0, v2 = 0;
#pragma unroll
    for (int v = 0; v < VPL; ++v) {             // first fill: everything is eligible
      const uint32_t c = uk[v];
      if (c > m1) { m2 = m1; v2 = v1; m1 = c; v1 = v; }
      else if (c > m2) { m2 = c; v2 = v; }
    }
    bool dry = false;                            // this lane has no expert left at all
    int my_id = 0;
    uint32_t my_key = 0;
    for (int j = 0; j < k; ++j) {
      const uint32_t gm = group_max_u32<LANES>(gmask, m1);
      const unsigned b = __ballot_sync(gmask, m1 == gm) & gmask;
      const int win = __ffs(b) - 1;
      const int id = __shfl_sync(gmask, e0 + v1, win);
      if (sub == j) { my_id = id; my_key = gm; }
      const bool iw = (lane == win);
      lk = iw ? m1 : lk;
      lv = iw ? v1 : lv;
      m1 = iw ? m2 : m1;
      v1 = iw ? v2 : v1;
      m2 = iw ? kTaken : m2;
      const bool need = (m1 == kTaken) && !dry;
      if (__any_sync(gmask, need)) {
        m1 = kTaken; m2 = kTaken; v1 = 0; v2 = 0;
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          const uint32_t c0 = uk[v];
          const bool elig = (c0 < lk) || (c0 == lk && v > lv);
          const uint32_t c = elig ? c0 : kTaken;
          if (c > m1) { m2 = m1; v2 = v1; m1 = c; v1 = v; }
          else if (c > m2) { m2 = c; v2 = v; }
        }
        dry = (m1 == kTaken);
      }
    }
    // the picked expert's logit: for softmax without groups the key IS the logit (-0 arrives as +0, same exp);
    // otherwise it is read back from the row (an L1/L2 hit, one load per pick): the sigmoid's key is not the logit,
    // and under a group limit a pick can come from a masked group (key -inf) when the kept groups hold fewer than k
    // experts that are not masked themselves (logits of -inf) -- its weight is that of its LOGIT (R1: weights from
    // the scores, the mask is selection-only)
    float my_x = 0.0f;
    if (sub < k) {
      if (SIGMOID || p.n_group > 1) my_x = __ldg(row + my_id);
      else my_x = __uint_as_float((my_key & 0x80000000u) ? (my_key & 0x7fffffffu) : ~my_key);
    }
    // ---- gate weights in fp64 for the picked experts (R1, R4, R5) ----
    double wj = 0.0;
    if (SIGMOID) {
      const double sj = (sub < k) ? 1.0 / (1.0 + exp(-(double)my_x)) : 0.0;
      wj = sj;
      if (p.renorm) wj = sj / group_sum_f64<LANES>(gmask, sj);
    } else {
      float lmx = x[0];
#pragma unroll
      for (int v = 1; v < VPL; ++v) lmx = fmaxf(lmx, x[v]);
      const float mx = __uint_as_float([](uint32_t o) { return (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o; }(
          group_max_u32<LANES>(gmask, ordered_u32(lmx))));
      const double ej = (sub < k) ? exp((double)my_x - (double)mx) : 0.0;
      double denom;
      if (p.renorm) {
        denom = group_sum_f64<LANES>(gmask, ej);
      } else {
        double part = 0.0;
#pragma unroll
        for (int v = 0; v < VPL; ++v) part += (e0 + v < E) ? (double)expf(x[v] - mx) : 0.0;
        denom = group_sum_f64<LANES>(gmask, part);
      }
      wj = ej / denom;
    }
    wj *= (double)p.scale;
    if (sub < k) {
      p.ids[(size_t)t * k + sub] = my_id;
      p.w[(size_t)t * k + sub] = __double2float_rn(wj);
      atomicAdd(&s_hist[my_id], 1);
    }
  }
  __syncthreads();
  ptx::griddep_wait();       // the kernel that zeroes the counts is the predecessor in the stream (see vibe_route_topk)
  for (int i = threadIdx.x; i < p.E; i += blockDim.x) {
    const int c = s_hist[i];
    if (c) atomicAdd(&p.counts[i], c);
  }
}


// ------------------------------------------------------------------------------------------------------------
// Wide-lane variant for E = 8 * VPL experts (VPL = 16 | 32: the 128- and 256-expert configs): one token per 8-lane
// group, FOUR tokens per warp, every lane owns VPL CONSECUTIVE experts (so lane order = expert order and the
// ballot's lowest lane is the lowest index among equal keys, as above).  Every warp-wide instruction of the
// selection rounds (redux, ballot, shuffle) now serves four tokens, and a lane keeps its first FOUR candidates in
// pick order (key, index) sorted in registers: a lane gives away more than four of a token's k <= 8 picks about
// once in a thousand tokens (then it rebuilds its heads from its registers).  ncu at 64K tokens x 256 experts, top-8:
// see profiles/r2_route_ncu.md (the 32-lane kernel needed 702 warp-instructions per token).
// Group-limited routing is supported when a group is exactly one lane's experts (n_group = 8: DeepSeek-V3's 8
// groups of 32): the group score is the lane's own top-2 sum, no cross-lane merge.
// ------------------------------------------------------------------------------------------------------------
#ifndef ROUTE8_MIN_BLOCKS
#define ROUTE8_MIN_BLOCKS 4
#endif
template <int VPL, bool SIGMOID>
__global__ void __launch_bounds__(256, ROUTE8_MIN_BLOCKS) route_topk8_kernel(const RouteParams p) {
  extern __shared__ int s_mem[];
  int* s_hist = s_mem;
  float* s_bias = reinterpret_cast<float*>(s_mem + p.E);      // [8][VPL + 1]: lane-major, padded (conflict-free)
  for (int i = threadIdx.x; i < p.E; i += blockDim.x) {
    s_hist[i] = 0;
    if (SIGMOID) s_bias[(i / VPL) * (VPL + 1) + i % VPL] = p.bias != nullptr ? p.bias[i] : 0.0f;
  }
  __syncthreads();
  constexpr int LANES = 8;
  const int lane = threadIdx.x & 31;
  const int sub = lane & 7;
  // Every collective below is issued with the FULL warp mask and stays inside the 8-lane groups by construction
  // (xor-shuffles with offsets 1, 2, 4; a full ballot of which each group reads its own byte; indexed shuffles with
  // a source lane of the own group): one instruction then serves the four tokens of the warp.  The same operations
  // with a per-group member mask execute once per distinct mask -- four times -- which is what made a first version
  // of this kernel slower than the 32-lane one.
  constexpr unsigned FULL = 0xffffffffu;
  const int gbase = lane & ~7;
  auto gmax_u32 = [&](uint32_t v) {
    v = max(v, __shfl_xor_sync(FULL, v, 1));
    v = max(v, __shfl_xor_sync(FULL, v, 2));
    return max(v, __shfl_xor_sync(FULL, v, 4));
  };
  auto gsum_f64 = [&](double v) {
    v += __shfl_xor_sync(FULL, v, 4);
    v += __shfl_xor_sync(FULL, v, 2);
    return v + __shfl_xor_sync(FULL, v, 1);
  };
  const int gidx = threadIdx.x >> 3;
  const int e0 = sub * VPL;
  const int E = p.E, k = p.k;
  const float NEG_INF = __int_as_float(0xff800000);

  const float* my_bias = s_bias + sub * (VPL + 1);
  auto unordered = [](uint32_t o) { return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o); };

  // the trip count is WARP-uniform (full-mask collectives inside): a group past the last token works on a copy of
  // token T-1 and stores nothing
  // (tiles of four tokens, interleaved over (warp, block): a last, partial round of tiles is spread over all blocks)
  const int n_tiles = (p.T + 3) >> 2;
  for (int tile = (threadIdx.x >> 5) * gridDim.x + blockIdx.x; tile < n_tiles; tile += 8 * gridDim.x) {
    const int tw = tile * 4;
    const bool valid = tw + (gidx & 3) < p.T;
    const int t = valid ? tw + (gidx & 3) : p.T - 1;
    // a lane's VPL * 4 bytes are contiguous: both 16-byte halves of every 32-byte sector are this lane's, read by
    // consecutive instructions, so the loads allocate in L1 (the second half is then an L1 hit, not a second L2 request)
    // Only the ordered keys stay in registers (the logits are recovered from them where the softmax needs them:
    // the map is a bijection up to -0 -> +0, which exp does not see).
    uint32_t uk[VPL];
    const uint4* row4 = reinterpret_cast<const uint4*>(p.logits + (size_t)t * E + e0);
#pragma unroll
    for (int q = 0; q < VPL / 4; ++q) {
      const uint4 u = __ldg(row4 + q);
      const float xv[4] = {__uint_as_float(u.x), __uint_as_float(u.y), __uint_as_float(u.z), __uint_as_float(u.w)};
#pragma unroll
      for (int c = 0; c < 4; ++c)
        uk[4 * q + c] = SIGMOID ? ordered_u32(__fadd_rn(vsig(xv[c]), my_bias[4 * q + c])) : ordered_u32(xv[c]);
    }
    // ---- sorted first four (key, index) of this lane; strict > keeps the lower index first among equal keys ----
    uint32_t h0 = kTaken, h1 = kTaken, h2 = kTaken, h3 = kTaken;
    int i0 = 0, i1 = 0, i2 = 0, i3 = 0;
    auto insert = [&](uint32_t c, int v) {
      const bool b0 = c > h0, b1 = c > h1, b2 = c > h2, b3 = c > h3;
      h3 = b2 ? h2 : (b3 ? c : h3);
      i3 = b2 ? i2 : (b3 ? v : i3);
      h2 = b1 ? h1 : (b2 ? c : h2);
      i2 = b1 ? i1 : (b2 ? v : i2);
      h1 = b0 ? h0 : (b1 ? c : h1);
      i1 = b0 ? i0 : (b1 ? v : i1);
      h0 = b0 ? c : h0;
      i0 = b0 ? v : i0;
    };
#pragma unroll
    for (int v = 0; v < VPL; ++v) insert(uk[v], v);
    // ---- group-limited routing (R6), one group per lane: score = sum of the lane's two largest keys ----
    if (p.n_group > 1) {
      const float k0 = unordered(h0);
      const float k1 = unordered(h1);
      const float score = (VPL >= 2) ? __fadd_rn(k0, k1) : k0;
      int rank = 0;
#pragma unroll
      for (int g2 = 0; g2 < LANES; ++g2) {
        const float s2 = __shfl_sync(FULL, score, gbase + g2);
        rank += (s2 > score || (s2 == score && g2 < sub)) ? 1 : 0;
      }
      if (rank >= p.topk_group) {
        const uint32_t ninf = ordered_u32(NEG_INF);
#pragma unroll
        for (int v = 0; v < VPL; ++v) uk[v] = ninf;
        h0 = h1 = h2 = h3 = ninf;      // indices 0..3 in order: still the lane's first four in pick order
        i0 = 0; i1 = 1; i2 = 2; i3 = 3;
      }
    }
    // ---- k rounds: redux-max over the lane heads, ballot, lowest lane wins, pop in the winner ----
    uint32_t lk = 0xffffffffu;
    int lv = -1;
    bool dry = false;
    int my_id = 0;
    uint32_t my_key = 0;
    for (int j = 0; j < k; ++j) {
      const uint32_t gm = gmax_u32(h0);
      const unsigned b = (__ballot_sync(FULL, h0 == gm) >> gbase) & 0xffu;
      const int win = gbase + __ffs(b) - 1;
      const int id = __shfl_sync(FULL, e0 + i0, win);
      if (sub == j) { my_id = id; my_key = gm; }
      if (lane == win) {
        lk = h0; lv = i0;
        h0 = h1; i0 = i1; h1 = h2; i1 = i2; h2 = h3; i2 = i3; h3 = kTaken;
      }
      const bool need = (h0 == kTaken) && !dry;
      if (__any_sync(FULL, need)) {            // rare: this lane gave away all four heads -> rebuild after (lk, lv)
        h0 = h1 = h2 = h3 = kTaken;
        i0 = i1 = i2 = i3 = 0;
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          const uint32_t c0 = uk[v];
          const bool elig = (c0 < lk) || (c0 == lk && v > lv);
          insert(elig ? c0 : kTaken, v);
        }
        dry = (h0 == kTaken);
      }
    }
    const float* row = p.logits + (size_t)t * E;
    float my_x = 0.0f;
    if (sub < k) {
      if (SIGMOID) my_x = __ldg(row + my_id);
      else my_x = unordered(my_key);
    }
    // ---- gate weights in fp64 for the picked experts (R1, R4, R5) ----
    double wj = 0.0;
    if (SIGMOID) {
      const double sj = (sub < k) ? 1.0 / (1.0 + exp(-(double)my_x)) : 0.0;
      wj = sj;
      if (p.renorm) wj = sj / gsum_f64(sj);
    } else {
      uint32_t lmx = uk[0];                    // (not h0: the heads have been popped)
#pragma unroll
      for (int v = 1; v < VPL; ++v) lmx = max(lmx, uk[v]);
      const float mx = unordered(gmax_u32(lmx));
      const double ej = (sub < k) ? exp((double)my_x - (double)mx) : 0.0;
      double denom;
      if (p.renorm) {
        denom = gsum_f64(ej);
      } else {
        double part = 0.0;
#pragma unroll
        for (int v = 0; v < VPL; ++v) part += (double)expf(unordered(uk[v]) - mx);
        denom = gsum_f64(part);
      }
      wj = ej / denom;
    }
    wj *= (double)p.scale;
    if (sub < k && valid) {
      p.ids[(size_t)t * k + sub] = my_id;
      p.w[(size_t)t * k + sub] = __double2float_rn(wj);
      atomicAdd(&s_hist[my_id], 1);
    }
  }
  __syncthreads();
  ptx::griddep_wait();       // the kernel that zeroes the counts is the predecessor in the stream (see vibe_route_topk)
  for (int i = threadIdx.x; i < p.E; i += blockDim.x) {
    const int c = s_hist[i];
    if (c) atomicAdd(&p.counts[i], c);
  }
}


// ------------------------------------------------------------------------------------------------------------
// Packed-key variant of the wide-lane kernel (no groups or 8 groups = one lane's experts each; sigmoid, or softmax
// with renormalisation: the two cases whose gate weights need the picked logits only).  ncu of route_topk8_kernel at 64K x 256 (profiles/
// r2_route_ncu.md): 390 warp-instructions per token, three quarters of them on the ALU pipe (ISETP/SEL/LOP3/VIMNMX:
// one warp-instruction per two cycles), most of them the (key, index) pairs dragged through the per-lane sorted
// insertion and the k selection rounds.  Here a key is ONE register: the order-preserving u32 image of the f32 key
// with its low 8 bits replaced by 255 - expert index, so keys are unique and ties go to the lowest index by
// construction.  A lane's first four (and its fifth) come out of min/max sorting networks, the group's first eight
// out of a three-level bitonic merge tree over the 8 lanes (20 shuffles, no ballot / find-first / indexed shuffle,
// no rounds), and the winners' indices out of the keys.
// The packed order differs from the exact one only between keys that agree in their upper 24 bits without being
// equal.  The tree leaves the picks in packed order and a bound on every key that was not picked (what its
// half-cleaners dropped and the lanes' fifths); if all adjacent pairs of {picks, bound} differ in the upper 24 bits,
// every pick is strictly above every other key of the token in exact order too and the result is exact.  Otherwise
// (about 3 tokens in 1000 on continuous f32 logits) the lanes OR the raw bits of the token's keys: if the low bytes
// of ALL keys are zero (bf16- or fp16-valued logits, where exact ties are common), equal upper bits mean equal keys
// and the packed tie-break is the exact one; else the token is redone by route_exact_token (one token per warp on
// exact keys).  A token of which one lane holds five or more picks (its fifth is above the last pick: 1 in 100)
// is redone the same way.
// The kernel is bound by the ALU pipe (about 520 of its 800 warp-instructions per 4-token tile).  What surrounds the
// arithmetic is arranged so that the pipe stays busy: the logits of a warp's next tile arrive by a bulk copy while it
// works on the current one, one block per SM hands tiles to its warps on demand, and the zeroing of the counts
// overlaps the kernel (programmatic dependent launch).  64K tokens x 256 experts, top-8: 44.0 -> 23 us.
// ------------------------------------------------------------------------------------------------------------
#define VIBE_CSWAP(a, b)                     \
  {                                          \
    const uint32_t hi_ = max(a, b);          \
    const uint32_t lo_ = min(a, b);          \
    a = hi_;                                 \
    b = lo_;                                 \
  }

// One token by one warp on the EXACT keys (32 lanes x E/32 consecutive experts, k rounds of {lane best, redux max,
// ballot, lowest lane wins}): the packed-key kernel calls it for the few tokens whose packed order is not provably the
// exact one.  Writes the token's ids / weights and counts it in the block histogram.  No groups or 8 groups of 4 lanes; sigmoid, or
// softmax with renormalisation (the configurations of the packed-key kernel).
// (h0..h3) sorted descending <- the four largest of (h0..h3) sorted and (a, b, c, d) in any order (sort the four, half-
// cleaner of the bitonic sequence h0 h1 h2 h3 d c b a, bitonic sort of the four kept); r5 <- the largest key seen so
// far that is not among them (the lane's fifth)
__device__ __forceinline__ void merge_quad5(uint32_t& h0, uint32_t& h1, uint32_t& h2, uint32_t& h3, uint32_t& r5, uint32_t a,
                                            uint32_t b, uint32_t c, uint32_t d) {
  VIBE_CSWAP(a, b);
  VIBE_CSWAP(c, d);
  VIBE_CSWAP(a, c);
  VIBE_CSWAP(b, d);
  VIBE_CSWAP(b, c);          // a >= b >= c >= d
  r5 = __vimax3_u32(r5, min(h0, d), min(h1, c));
  r5 = __vimax3_u32(r5, min(h2, b), min(h3, a));
  h0 = max(h0, d);
  h1 = max(h1, c);
  h2 = max(h2, b);
  h3 = max(h3, a);
  VIBE_CSWAP(h0, h2);
  VIBE_CSWAP(h1, h3);
  VIBE_CSWAP(h0, h1);
  VIBE_CSWAP(h2, h3);
}
// one step of the cross-lane merge tree: against the partner's (q0..q3) the lane keeps the larger (or, low = true, the
// smaller) of every pair -- a bitonic four -- and sorts them
__device__ __forceinline__ void tree_exchange(uint32_t& h0, uint32_t& h1, uint32_t& h2, uint32_t& h3, uint32_t q0, uint32_t q1,
                                              uint32_t q2, uint32_t q3, bool low) {
  h0 = low ? min(h0, q0) : max(h0, q0);
  h1 = low ? min(h1, q1) : max(h1, q1);
  h2 = low ? min(h2, q2) : max(h2, q2);
  h3 = low ? min(h3, q3) : max(h3, q3);
  VIBE_CSWAP(h0, h2);
  VIBE_CSWAP(h1, h3);
  VIBE_CSWAP(h0, h1);
  VIBE_CSWAP(h2, h3);
}
// half-cleaner against the partner's reversed four: keep the larger of every pair, remember the largest dropped key
__device__ __forceinline__ void tree_halfclean(uint32_t& h0, uint32_t& h1, uint32_t& h2, uint32_t& h3, uint32_t& dmax,
                                               uint32_t q0, uint32_t q1, uint32_t q2, uint32_t q3) {
  dmax = __vimax3_u32(dmax, min(h0, q0), min(h1, q1));
  dmax = __vimax3_u32(dmax, min(h2, q2), min(h3, q3));
  h0 = max(h0, q0);
  h1 = max(h1, q1);
  h2 = max(h2, q2);
  h3 = max(h3, q3);
}

template <int VPL, bool SIGMOID, bool GROUPED>
__device__ __noinline__ void route_exact_token(const float* logits, int32_t* ids, float* w, int k, int renorm, float scale,
                                               int topk_group, int t, int* s_hist, const float* s_bias) {
  constexpr int E = 8 * VPL;
  constexpr int V = E / 32;
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const float* row = logits + (size_t)t * E;
  uint32_t uk[V];
  float fk[V];
#pragma unroll
  for (int q = 0; q < V / 4; ++q) {
    const uint4 u = __ldg(reinterpret_cast<const uint4*>(row + lane * V) + q);
    const float xv[4] = {__uint_as_float(u.x), __uint_as_float(u.y), __uint_as_float(u.z), __uint_as_float(u.w)};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int e = lane * V + 4 * q + c;
      const float key = SIGMOID ? __fadd_rn(vsig(xv[c]), s_bias[(e / VPL) * (VPL + 1) + e % VPL]) : xv[c];
      fk[4 * q + c] = key;
      uk[4 * q + c] = ordered_u32(key);
    }
  }
  if (GROUPED) {
    // 8 groups of VPL consecutive experts = 4 lanes each: score = sum of the group's two largest keys (R6)
    const float NEG_INF = __int_as_float(0xff800000);
    float m1 = NEG_INF, m2 = NEG_INF;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const float c = fk[v];
      if (c > m1) { m2 = m1; m1 = c; } else if (c > m2) { m2 = c; }
    }
#pragma unroll
    for (int o = 1; o < 4; o <<= 1) {
      const float q1 = __shfl_xor_sync(FULL, m1, o);
      const float q2 = __shfl_xor_sync(FULL, m2, o);
      const float lo = fminf(m1, q1);
      m1 = fmaxf(m1, q1);
      m2 = fmaxf(lo, fmaxf(m2, q2));
    }
    const float score = __fadd_rn(m1, m2);
    const int g = lane >> 2;
    int rank = 0;
#pragma unroll
    for (int g2 = 0; g2 < 8; ++g2) {
      const float s2 = __shfl_sync(FULL, score, g2 * 4);
      rank += (s2 > score || (s2 == score && g2 < g)) ? 1 : 0;
    }
    if (rank >= topk_group) {
#pragma unroll
      for (int v = 0; v < V; ++v) uk[v] = ordered_u32(NEG_INF);
    }
  }
  int my_id = 0;
  for (int j = 0; j < k; ++j) {
    uint32_t best = kTaken;
    int bv = 0;
#pragma unroll
    for (int v = 0; v < V; ++v)
      if (uk[v] > best) { best = uk[v]; bv = v; }
    const uint32_t gm = __reduce_max_sync(FULL, best);
    const int win = __ffs(__ballot_sync(FULL, best == gm)) - 1;
    const int id = __shfl_sync(FULL, lane * V + bv, win);
    if (lane == j) my_id = id;
    if (lane == win) {
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (v == bv) uk[v] = kTaken;
    }
  }
  auto wsum_f64 = [&](double v) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
  };
  const float my_x = (lane < k) ? __ldg(row + my_id) : 0.0f;
  double wj;
  if (SIGMOID) {
    const double sj = (lane < k) ? 1.0 / (1.0 + exp(-(double)my_x)) : 0.0;
    wj = sj;
    if (renorm) wj = sj / wsum_f64(sj);
  } else {
    const float mx = __shfl_sync(FULL, my_x, 0);
    const double ej = (lane < k) ? exp((double)my_x - (double)mx) : 0.0;
    wj = ej / wsum_f64(ej);
  }
  wj *= (double)scale;
  if (lane < k) {
    ids[(size_t)t * k + lane] = my_id;
    w[(size_t)t * k + lane] = __double2float_rn(wj);
    atomicAdd(&s_hist[my_id], 1);
  }
}

// shared memory of route_topk8p_kernel: histogram, padded bias, then (128-byte aligned) one 4-token staging buffer and
// one mbarrier per warp, then the block's tile counter
#ifndef ROUTE8P_WARPS_N
#define ROUTE8P_WARPS_N 28
#endif
constexpr int ROUTE8P_REDO_CAP = 126;   // tokens a block may put off to its end (more are redone on the spot)
constexpr int ROUTE8P_WARPS = ROUTE8P_WARPS_N;      // ONE block of up to 28 warps per SM (72 registers per thread; with 32 warps of 64 registers the merge networks spill)
template <int VPL>
__host__ __device__ constexpr size_t route8p_stage_off(bool sigmoid) {
  return ((size_t)8 * VPL * sizeof(int) + (sigmoid ? (size_t)8 * (VPL + 1) * sizeof(float) : 0) + 127) & ~(size_t)127;
}
template <int VPL>
__host__ __device__ constexpr size_t route8p_smem_bytes(bool sigmoid, int warps) {
  return route8p_stage_off<VPL>(sigmoid) + (size_t)warps * 4 * 8 * VPL * sizeof(float) + warps * sizeof(uint64_t) +
         (2 + ROUTE8P_REDO_CAP) * sizeof(int) + 8;
}

template <int VPL, bool SIGMOID, bool GROUPED>
__global__ void __launch_bounds__(ROUTE8P_WARPS * 32, 1) route_topk8p_kernel(const RouteParams p) {
  const int NW = blockDim.x >> 5;
  extern __shared__ __align__(128) int s_mem[];
  constexpr int E = 8 * VPL;
  constexpr uint32_t TILE_BYTES = 4u * E * sizeof(float);
  int* s_hist = s_mem;
  float* s_bias = reinterpret_cast<float*>(s_mem + E);        // [8][VPL + 1]: lane-major, padded (conflict-free)
  char* s_stage = reinterpret_cast<char*>(s_mem) + route8p_stage_off<VPL>(SIGMOID);
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t my_stage = ptx::smem_u32(s_stage + (size_t)warp * TILE_BYTES);
  const uint32_t my_bar = ptx::smem_u32(s_stage + (size_t)NW * TILE_BYTES + (size_t)warp * sizeof(uint64_t));
  // The logits of a warp's NEXT tile (four consecutive tokens: 4 KB / 2 KB contiguous) are fetched by one bulk copy
  // into the warp's staging buffer while the warp works on the current tile from registers: the DRAM latency, which
  // the 64-register / 8-warps-per-scheduler budget cannot hide with loads into registers, is off the critical path.
  const int n_tiles = (p.T + 3) >> 2;
  auto fetch = [&](int tile) {
    const int ntok = min(4, p.T - tile * 4);
    const uint32_t bytes = (uint32_t)ntok * E * (uint32_t)sizeof(float);
    ptx::mbar_arrive_expect_tx(my_bar, bytes);
    ptx::bulk_load_1d(my_stage, p.logits + (size_t)tile * 4 * E, bytes, my_bar);
  };
  // Tiles of four tokens; block b (one per SM) owns tiles b, b + G, b + 2G, ... (G = grid size) and hands them to its
  // warps on demand (shared counter): a warp that had to redo tokens on exact keys, or that the scheduler served
  // less often, simply takes fewer tiles, and all warps of the SM end together.  With a static
  // assignment to four blocks of 8 warps per SM the blocks of one SM ended between 12 and 27 us of a 30 us kernel
  // (64K tokens x 256 experts, in-kernel timestamps).
  int* s_next = reinterpret_cast<int*>(s_stage + (size_t)NW * TILE_BYTES + NW * sizeof(uint64_t));
  // s_next[1]: number of, s_next[2..]: the tokens whose exact redo was put off to the end of the block (see below)
  int* s_redo_n = s_next + 1;
  int* s_redo = s_next + 2;
  if (threadIdx.x == 0) {
    *s_next = NW;
    *s_redo_n = 0;
  }
  int tile = warp * gridDim.x + blockIdx.x;
  if (lane == 0) {
    ptx::mbar_init(my_bar, 1);
    ptx::fence_barrier_init();
    if (tile < n_tiles) fetch(tile);
  }
  for (int i = threadIdx.x; i < E; i += blockDim.x) {
    s_hist[i] = 0;
    if (SIGMOID) s_bias[(i / VPL) * (VPL + 1) + i % VPL] = p.bias != nullptr ? p.bias[i] : 0.0f;
  }
  __syncthreads();
  constexpr unsigned FULL = 0xffffffffu;       // full-mask collectives that stay inside the 8-lane groups (see above)
  const int sub = lane & 7;
  const int gbase = lane & ~7;
  auto gmax_u32 = [&](uint32_t v) {
    v = max(v, __shfl_xor_sync(FULL, v, 1));
    v = max(v, __shfl_xor_sync(FULL, v, 2));
    return max(v, __shfl_xor_sync(FULL, v, 4));
  };
  auto gsum_f64 = [&](double v) {
    v += __shfl_xor_sync(FULL, v, 4);
    v += __shfl_xor_sync(FULL, v, 2);
    return v + __shfl_xor_sync(FULL, v, 1);
  };
  // Which experts a lane holds.  GROUPED: VPL consecutive ones (a group is one lane's experts).  Otherwise the
  // 16-byte chunks of the row are dealt round the 8 lanes -- chunk q * 8 + sub at step q, experts 32 q + 4 sub + c:
  // the 8 lanes of a token read 128 contiguous bytes of the staged row (no bank conflict, no rotation), and the
  // index byte of a key is a compile-time constant (255 - 32 q - c, inserted by one PRMT) less the lane's 4 sub,
  // which comes off the five survivors of the network instead of off all VPL keys.
  const uint32_t e0 = GROUPED ? (uint32_t)(sub * VPL) : (uint32_t)(4 * sub);
  const int k = p.k;
  const float* my_bias = s_bias + sub * (VPL + 1);
  const float* il_bias = s_bias + (VPL == 32 ? 4 * sub : (sub >= 4 ? 4 * sub + 1 : 4 * sub));     // interleaved mapping: see below
  // f32 key -> order-preserving u32 with the low byte set (the caller subtracts the index): -0 -> +0 first
  auto packed_hi = [](float key) {
    const uint32_t b = __float_as_uint(__fadd_rn(key, 0.0f));
    const uint32_t t = (uint32_t)((int32_t)b >> 31) | 0x80000000u;
    return (b ^ t) | 0xffu;
  };
  // Sigmoid keys are APPROXIMATE here (2 MUFU + 3 FMA-pipe operations instead of the ~25 separately rounded ones of
  // vsig): |approx - vsig| < 2^-21 (ex2.approx 2^-22 and rcp.approx 2^-23 relative; vsig itself is within 1.2e-7 of
  // the sigmoid), the keys (+ bias, rounded) differ by that and one ulp at most.  For keys >= 2^-4 one unit of the
  // upper 24 bits is >= 2^-19, and two keys whose upper 24 bits are two or more units apart differ by more than one
  // unit: they are in the same order exactly as approximately.  Wherever the selection leans on a
  // smaller gap (or on a key below 2^-4) the token is redone on exact keys; the group scores use exact keys of the
  // two candidates.
  auto approx_sig = [](float x) {
    float e, r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * -1.44269504f));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + e));
    return r;
  };
  constexpr uint32_t GAP_MIN = SIGMOID ? 2u : 1u;
  constexpr uint32_t PK_FLOOR = 0xbd800000u;     // order-preserving image of 2^-4 (0x3d800000 | sign bit)
  // a lane's VPL consecutive experts are CH 16-byte chunks of the staged row; the lanes of a quarter-warp read them
  // in rotated order (chunk (q + rot) mod CH at step q), which spreads the 8 lanes over all 32 banks
  constexpr int CH = VPL / 4;
  const int rot = sub / (8 / CH);
  const uint4* my_row4 = reinterpret_cast<const uint4*>(s_stage + (size_t)warp * TILE_BYTES) + (lane >> 3) * (E / 4) +
                         (GROUPED ? sub * CH : sub);

  uint32_t phase = 0;
  while (tile < n_tiles) {
    const int tbase = tile * 4;
    const int tt = tbase + (lane >> 3);
    const bool valid = tt < p.T;
    const int t = valid ? tt : p.T - 1;
    const float* row = p.logits + (size_t)t * E;
    uint32_t pk[VPL];                          // packed keys with the IN-LANE index (low byte 255 - v)
    ptx::mbar_wait(my_bar, phase);
    phase ^= 1u;
    if (GROUPED) {
#pragma unroll
      for (int q = 0; q < CH; ++q) {
        const int ch = (q + rot) & (CH - 1);
        const uint4 u = my_row4[ch];
        const float xv[4] = {__uint_as_float(u.x), __uint_as_float(u.y), __uint_as_float(u.z), __uint_as_float(u.w)};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const float key = SIGMOID ? __fadd_rn(approx_sig(xv[c]), my_bias[4 * ch + c]) : xv[c];
          pk[4 * q + c] = packed_hi(key) - (uint32_t)(4 * ch) - (uint32_t)c;
        }
      }
    } else {
#pragma unroll
      for (int q = 0; q < CH; ++q) {
        const uint4 u = my_row4[q * 8];
        const float xv[4] = {__uint_as_float(u.x), __uint_as_float(u.y), __uint_as_float(u.z), __uint_as_float(u.w)};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          // (the bias of expert e = 32 q + 4 sub + c in the padded [8][VPL + 1] layout)
          const int eb = 32 * q + c;                                     // + 4 sub
          const float key = SIGMOID ? __fadd_rn(approx_sig(xv[c]), il_bias[(eb / VPL) * (VPL + 1) + eb % VPL]) : xv[c];
          const uint32_t bq = __float_as_uint(__fadd_rn(key, 0.0f));
          const uint32_t tq = (uint32_t)((int32_t)bq >> 31) | 0x80000000u;
          pk[4 * q + c] = __byte_perm(bq ^ tq, 255u - (uint32_t)(32 * q + c), 0x3214);
        }
      }
    }
    // every lane has consumed its part of the buffer: the next tile's copy may overwrite it
    __syncwarp();
    {
      int nxt = 0;
      if (lane == 0) {
        nxt = atomicAdd(s_next, 1) * (int)gridDim.x + (int)blockIdx.x;
        if (nxt < n_tiles) fetch(nxt);
      }
      tile = __shfl_sync(FULL, nxt, 0);      // (the rest of this iteration addresses its tile through t / row only)
    }
    // ---- the lane's four largest, sorted, and its fifth (r5); then the lane's first expert goes into the index byte ----
    uint32_t h0 = 0, h1 = 0, h2 = 0, h3 = 0, r5 = 0;
#pragma unroll
    for (int q = 0; q < VPL / 4; ++q)
      merge_quad5(h0, h1, h2, h3, r5, pk[4 * q], pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
    bool unsure = false;                       // this lane's part of "the packed order may not be the exact one"
    if (GROUPED) {
      // ---- group-limited routing (R6), one group per lane: score = sum of the lane's two largest EXACT keys.  The
      //      two are the first two of the packed order if the second is clear of the third (margin below). ----
      unsure = (h1 >> 8) - (h2 >> 8) < GAP_MIN || (SIGMOID && h1 < PK_FLOOR);
      const int v0 = 255 - (int)(h0 & 0xffu), v1 = 255 - (int)(h1 & 0xffu);
      float k0 = __ldg(row + e0 + v0), k1 = __ldg(row + e0 + v1);
      if (SIGMOID) {
        k0 = __fadd_rn(vsig(k0), my_bias[v0]);
        k1 = __fadd_rn(vsig(k1), my_bias[v1]);
      }
      const float score = __fadd_rn(k0, k1);
      int rank = 0;
#pragma unroll
      for (int g2 = 0; g2 < 8; ++g2) {
        const float s2 = __shfl_sync(FULL, score, gbase + g2);
        rank += (s2 > score || (s2 == score && g2 < sub)) ? 1 : 0;
      }
      if (rank >= p.topk_group) { h0 = h1 = h2 = h3 = r5 = e0; }     // (e0 is subtracted below: the group is out)
    }
    h0 -= e0; h1 -= e0; h2 -= e0; h3 -= e0; r5 -= e0;
    // ---- the group's eight largest heads by a bitonic merge tree over the 8 lanes (three levels) ----
    // Level L merges the sorted 8 of two 2^(L-1)-lane halves: half-cleaner against the reversed partner list (all
    // lanes keep the larger: both halves then hold the 8 largest, as mirrored copies), one exchange between the lane
    // with the upper and the lane with the lower four, a local bitonic sort.  After level 3 the lanes of even parity
    // (0, 3, 5, 6) hold picks 1..4 and those of odd parity (1, 2, 4, 7) picks 5..8, sorted, in h0..h3.  What the
    // half-cleaners drop, and the lanes' fifths, bound everything that was not picked (dmax).
    uint32_t dmax = r5;
    {
      const bool low1 = (sub & 1) != 0;
      tree_exchange(h0, h1, h2, h3, __shfl_xor_sync(FULL, h3, 1), __shfl_xor_sync(FULL, h2, 1),
                    __shfl_xor_sync(FULL, h1, 1), __shfl_xor_sync(FULL, h0, 1), low1);
      const bool low2 = (__popc(sub & 3) & 1) != 0;
      tree_halfclean(h0, h1, h2, h3, dmax, __shfl_xor_sync(FULL, h3, 3), __shfl_xor_sync(FULL, h2, 3),
                     __shfl_xor_sync(FULL, h1, 3), __shfl_xor_sync(FULL, h0, 3));
      tree_exchange(h0, h1, h2, h3, __shfl_xor_sync(FULL, h0, 1), __shfl_xor_sync(FULL, h1, 1),
                    __shfl_xor_sync(FULL, h2, 1), __shfl_xor_sync(FULL, h3, 1), low2);
      tree_halfclean(h0, h1, h2, h3, dmax, __shfl_xor_sync(FULL, h3, 5), __shfl_xor_sync(FULL, h2, 5),
                     __shfl_xor_sync(FULL, h1, 5), __shfl_xor_sync(FULL, h0, 5));
    }
    const bool low3 = (__popc(sub) & 1) != 0;
    tree_exchange(h0, h1, h2, h3, __shfl_xor_sync(FULL, h0, 1), __shfl_xor_sync(FULL, h1, 1),
                  __shfl_xor_sync(FULL, h2, 1), __shfl_xor_sync(FULL, h3, 1), low3);
    // this lane's pick: number myj in the order of the picks
    const int slot = sub >> 1;
    const int myj = (low3 ? 4 : 0) + slot;
    const uint32_t my_p = slot == 0 ? h0 : slot == 1 ? h1 : slot == 2 ? h2 : h3;
    int my_id = 255 - (int)(my_p & 0xffu);
    bool redo = false;
    // ---- is the packed order the exact one?  the picks and the best key that was not picked must differ in their
    //      upper 24 bits; a key above the last pick that was not picked (a lane with five or more of the picks: its
    //      heads ran out) sends the token to the exact routine too ----
    {
      const uint32_t rest = gmax_u32(dmax);
      const uint32_t cross = __shfl_xor_sync(FULL, h0, 1);             // an upper lane reads pick 5 here
      uint32_t nxt = slot == 0 ? h1 : slot == 1 ? h2 : slot == 2 ? h3 : (low3 ? 0u : cross);
      if (myj == k - 1) nxt = max(nxt, rest);
      // exact keys (softmax): equal upper 24 bits; approximate keys (sigmoid, error far below one unit of the upper
      // 24 bits for keys >= 2^-4): less than two units apart, or a last pick below 2^-4
      const bool ran_out = (myj == k - 1) && nxt > my_p;
      const bool close = SIGMOID ? (my_p >> 8) - (nxt >> 8) < GAP_MIN : (my_p ^ nxt) < 256u;
      const bool collide = (myj < k) && (close || nxt > my_p || (SIGMOID && myj == k - 1 && my_p < PK_FLOOR));
      const unsigned cb = __ballot_sync(FULL, collide || unsure);
      if (cb != 0u) {
        // softmax: equal upper bits are exact ties if the low bytes of all keys of the token are zero, else the token
        // is redone; a doubtful group score, a lane that ran out of heads or approximate keys: always redone
        bool hard = unsure || ran_out || (SIGMOID && collide);
        if (!SIGMOID) {
          uint32_t lo = 0;                       // OR of the raw bits of the lane's keys (reloaded: L2 hits)
          const uint4* grow4 = reinterpret_cast<const uint4*>(row + sub * VPL);      // (any partition of the row does)
#pragma unroll
          for (int q = 0; q < CH; ++q) {
            const uint4 u = __ldg(grow4 + q);
            lo |= u.x | u.y | u.z | u.w;
          }
          lo |= __shfl_xor_sync(FULL, lo, 1);
          lo |= __shfl_xor_sync(FULL, lo, 2);
          lo |= __shfl_xor_sync(FULL, lo, 4);
          hard = hard || (collide && (lo & 0xffu) != 0u);
        }
        const unsigned hb = __ballot_sync(FULL, hard);
        redo = ((hb >> gbase) & 0xffu) != 0u && valid;
        const unsigned rb = __ballot_sync(FULL, redo);
        // With several tiles per warp a token is redone on the spot (the other warps take the tiles this warp does
        // not, and a redo in a last tile overlaps the other warps' last tiles).  In a single-wave launch (one tile
        // per warp: all warps end together) the tokens are left to the block: after the loop every warp takes one,
        // side by side, instead of one warp holding the block's end back by two or three redos in a row
        // (C3, 16K tokens: 18.6 -> 14.5 us).
        // (softmax keys are exact and redone 1 token in 80: putting those off costs more than it saves -- measured)
        const bool last_tile = SIGMOID && n_tiles <= (int)gridDim.x * NW;
        for (int g = 0; g < 4; ++g)
          if ((rb >> (8 * g)) & 1u) {
            int slot = ROUTE8P_REDO_CAP;
            if (last_tile) {
              if (lane == 0) slot = atomicAdd(s_redo_n, 1);
              slot = __shfl_sync(FULL, slot, 0);
            }
            if (slot < ROUTE8P_REDO_CAP) {
              if (lane == 0) s_redo[slot] = tbase + g;
            } else {
              route_exact_token<VPL, SIGMOID, GROUPED>(p.logits, p.ids, p.w, k, p.renorm, p.scale, p.topk_group, tbase + g, s_hist, s_bias);
            }
          }
      }
    }
    // ---- gate weights in fp64 for the picked experts (R1, R4, R5) ----
    const float my_x = (myj < k) ? __ldg(row + my_id) : 0.0f;
    double wj;
    if (SIGMOID) {
      const double sj = (myj < k) ? 1.0 / (1.0 + exp(-(double)my_x)) : 0.0;
      wj = sj;
      if (p.renorm) wj = sj / gsum_f64(sj);
    } else {
      const float mx = __shfl_sync(FULL, my_x, gbase);      // the first pick (lane 0 of the group) is the row maximum
      const double ej = (myj < k) ? exp((double)my_x - (double)mx) : 0.0;
      wj = ej / gsum_f64(ej);                               // renormalised: the denominator over all experts cancels
    }
    wj *= (double)p.scale;
    if (myj < k && valid && !redo) {
      p.ids[(size_t)t * k + myj] = my_id;
      p.w[(size_t)t * k + myj] = __double2float_rn(wj);
      atomicAdd(&s_hist[my_id], 1);
    }
  }
  __syncthreads();
  {
    const int n_redo = min(*s_redo_n, ROUTE8P_REDO_CAP);
    for (int i = warp; i < n_redo; i += NW)
      route_exact_token<VPL, SIGMOID, GROUPED>(p.logits, p.ids, p.w, p.k, p.renorm, p.scale, p.topk_group, s_redo[i], s_hist, s_bias);
    if (n_redo > 0) __syncthreads();
  }
  ptx::griddep_wait();       // the kernel that zeroes the counts is the predecessor in the stream (see vibe_route_topk)
  for (int i = threadIdx.x; i < p.E; i += blockDim.x) {
    const int c = s_hist[i];
    if (c) atomicAdd(&p.counts[i], c);
  }
}

template <int VPL>
vibe_status launch_route8(const RouteParams& p, bool sigmoid, bool packed, cudaStream_t st) {
  // one resident wave (4 blocks of 8 warps per SM), tiles of four tokens interleaved over warps and blocks
  int blocks = ((p.T + 3) / 4 + 7) / 8;
  const int cap = num_sms() * ROUTE8_MIN_BLOCKS;
  if (blocks > cap) blocks = cap;
  const size_t smem = (size_t)p.E * sizeof(int) + (sigmoid ? (size_t)8 * (VPL + 1) * sizeof(float) : 0);
  if (packed) {
    const bool grouped = p.n_group > 1;
    static std::mutex mu;
    static bool done[kMaxDevices] = {};
    {
      std::lock_guard<std::mutex> lk(mu);
      const int dev = current_device();
      if (!done[dev]) {      // the opt-in to > 48 KB of dynamic shared memory is per device
        const int big = (int)route8p_smem_bytes<VPL>(true, ROUTE8P_WARPS);
        VIBE_CUDA(cudaFuncSetAttribute(route_topk8p_kernel<VPL, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
        VIBE_CUDA(cudaFuncSetAttribute(route_topk8p_kernel<VPL, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
        VIBE_CUDA(cudaFuncSetAttribute(route_topk8p_kernel<VPL, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
        VIBE_CUDA(cudaFuncSetAttribute(route_topk8p_kernel<VPL, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
        done[dev] = true;
      }
    }
    // one block per SM; a small batch is spread over all SMs with fewer warps per block
    const int n_tiles = (p.T + 3) / 4;
    int warps = (n_tiles + num_sms() - 1) / num_sms();
    warps = warps < 1 ? 1 : warps > ROUTE8P_WARPS ? ROUTE8P_WARPS : warps;
    int pblocks = (n_tiles + warps - 1) / warps;
    if (pblocks > num_sms()) pblocks = num_sms();
    const size_t psmem = route8p_smem_bytes<VPL>(sigmoid, warps);
    const dim3 pg(pblocks), pb(warps * 32);
    if (sigmoid && grouped)
      (void)launch_pdl(route_topk8p_kernel<VPL, true, true>, pg, pb, psmem, st, p);
    else if (sigmoid)
      (void)launch_pdl(route_topk8p_kernel<VPL, true, false>, pg, pb, psmem, st, p);
    else if (grouped)
      (void)launch_pdl(route_topk8p_kernel<VPL, false, true>, pg, pb, psmem, st, p);
    else
      (void)launch_pdl(route_topk8p_kernel<VPL, false, false>, pg, pb, psmem, st, p);
    VIBE_LAUNCH_CHECK("route_topk8p_kernel");
    return VIBE_OK;
  }
  if (sigmoid)
    (void)launch_pdl(route_topk8_kernel<VPL, true>, dim3(blocks), dim3(256), smem, st, p);
  else
    (void)launch_pdl(route_topk8_kernel<VPL, false>, dim3(blocks), dim3(256), smem, st, p);
  VIBE_LAUNCH_CHECK("route_topk8_kernel");
  return VIBE_OK;
}

template <int LANES, int VPL>
vibe_status launch_route(const RouteParams& p, bool sigmoid, cudaStream_t st) {
  constexpr int gpb = 256 / LANES;
  int blocks = (p.T + gpb - 1) / gpb;
  const int cap = num_sms() * 8;
  if (blocks > cap) blocks = cap;
  size_t smem = (size_t)p.E * sizeof(int);
  if (p.n_group > 1 && !p.fast_groups) smem += (size_t)gpb * p.n_group * sizeof(float);
  if (sigmoid)
    (void)launch_pdl(route_topk_kernel<LANES, VPL, true>, dim3(blocks), dim3(256), smem, st, p);
  else
    (void)launch_pdl(route_topk_kernel<LANES, VPL, false>, dim3(blocks), dim3(256), smem, st, p);
  VIBE_LAUNCH_CHECK("route_topk_kernel");
  return VIBE_OK;
}

}  // namespace
}  // namespace vibe

extern "C" vibe_status vibe_route_topk(const vibe_route_cfg* cfg, const float* logits, int32_t T, int32_t* topk_ids,
                                       float* topk_w, int32_t* counts, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_route_topk: cfg is NULL");
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_route_topk: need 1 <= k <= E (E=%d k=%d)", E, k);
  VIBE_REQUIRE(T >= 0, VIBE_ERR_INVALID_ARG, "vibe_route_topk: T < 0");
  VIBE_REQUIRE((int64_t)T * k < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "vibe_route_topk: T*k >= 2^31");
  VIBE_REQUIRE(cfg->score_fn == VIBE_SCORE_SOFTMAX || cfg->score_fn == VIBE_SCORE_SIGMOID, VIBE_ERR_INVALID_ARG,
               "vibe_route_topk: unknown score_fn %d", cfg->score_fn);
  VIBE_REQUIRE(counts != nullptr, VIBE_ERR_INVALID_ARG, "vibe_route_topk: counts is NULL");
  VIBE_REQUIRE(T == 0 || (logits && topk_ids && topk_w), VIBE_ERR_INVALID_ARG, "vibe_route_topk: NULL tensor");
  VIBE_REQUIRE(T == 0 || aligned16(logits), VIBE_ERR_INVALID_ARG, "vibe_route_topk: logits must be 16-byte aligned");
  const int ng = cfg->n_group > 1 ? cfg->n_group : 0;
  if (ng) {
    VIBE_REQUIRE(E % ng == 0, VIBE_ERR_INVALID_ARG, "vibe_route_topk: E %% n_group != 0");
    VIBE_REQUIRE(cfg->topk_group >= 1 && cfg->topk_group <= ng, VIBE_ERR_INVALID_ARG,
                 "vibe_route_topk: need 1 <= topk_group <= n_group");
    VIBE_REQUIRE((int64_t)cfg->topk_group * (E / ng) >= k, VIBE_ERR_INVALID_ARG,
                 "vibe_route_topk: topk_group * (E/n_group) < k");
  }
  VIBE_REQUIRE(E <= 512, VIBE_ERR_UNSUPPORTED, "vibe_route_topk: E > 512 not implemented");
  VIBE_REQUIRE(k <= 32, VIBE_ERR_UNSUPPORTED, "vibe_route_topk: k > 32 not implemented");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  route_zero_counts_kernel<<<1, 256, 0, st>>>(counts, E);
  VIBE_LAUNCH_CHECK("route_zero_counts_kernel");
  if (T == 0) return VIBE_OK;

  RouteParams p;
  p.logits = logits;
  p.bias = cfg->select_bias;
  p.ids = topk_ids;
  p.w = topk_w;
  p.counts = counts;
  p.T = T;
  p.E = E;
  p.k = k;
  p.renorm = cfg->renormalize ? 1 : 0;
  p.scale = cfg->routed_scale;
  p.n_group = ng;
  p.topk_group = cfg->topk_group;
  const bool sig = cfg->score_fn == VIBE_SCORE_SIGMOID;

  // 128 / 256 experts, top-k <= 8: four tokens per warp (route_topk8_kernel); group-limited only with 8 groups
  // (not the un-renormalised softmax with group limiting: the wide-lane kernel overwrites the keys of masked groups,
  // and that denominator runs over ALL logits; keeping them costs a register, a spill and 15 % of the kernel's speed
  // for every other configuration -- measured --, so this one combination takes the 32-lane kernel)
  if ((E == 128 || E == 256) && k <= 8 && (ng == 0 || (ng == 8 && (sig || cfg->renormalize)))) {
    p.fast_groups = 1;
    // packed one-register keys where the gate weights need the picked logits only (with or without the 8 groups);
    // route_topk8_kernel is left with the un-renormalised softmax without groups
    const bool packed = sig || cfg->renormalize;
    return E == 256 ? launch_route8<32>(p, sig, packed, st) : launch_route8<16>(p, sig, packed, st);
  }
  int lanes, vpl;
  if (E <= 64 && k <= 8) {
    lanes = 8;
    vpl = E <= 8 ? 1 : E <= 16 ? 2 : E <= 32 ? 4 : 8;
  } else {
    lanes = 32;
    vpl = E <= 32 ? 1 : E <= 64 ? 2 : E <= 128 ? 4 : E <= 256 ? 8 : 16;
  }
  p.fast_groups = 0;
  if (ng) {
    const int gs = E / ng;
    if (gs % vpl == 0) {
      const int lpg = gs / vpl;
      if ((lpg & (lpg - 1)) == 0 && lpg <= lanes) p.fast_groups = 1;
    }
    VIBE_REQUIRE(p.fast_groups || ng <= 64, VIBE_ERR_UNSUPPORTED,
                 "vibe_route_topk: n_group > 64 with irregular group size not implemented");
  }
#define VIBE_ROUTE_CASE(L, V) \
  if (lanes == L && vpl == V) return launch_route<L, V>(p, sig, st);
  VIBE_ROUTE_CASE(8, 1)
  VIBE_ROUTE_CASE(8, 2)
  VIBE_ROUTE_CASE(8, 4)
  VIBE_ROUTE_CASE(8, 8)
  VIBE_ROUTE_CASE(32, 1)
  VIBE_ROUTE_CASE(32, 2)
  VIBE_ROUTE_CASE(32, 4)
  VIBE_ROUTE_CASE(32, 8)
  VIBE_ROUTE_CASE(32, 16)
#undef VIBE_ROUTE_CASE
  set_error("vibe_route_topk: no kernel for E=%d k=%d", E, k);
  return VIBE_ERR_UNSUPPORTED;
}
