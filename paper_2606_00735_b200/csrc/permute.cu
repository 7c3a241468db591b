// permute.cu -- a3: stable counting sort of assignments by local expert slot + row gather
// (vibe_permute).  Semantics: include/vibe.h, readings P1-P4.
//
// Two launches on one stream, no host sync, no spin-waits between CTAs.  The batch is cut
// into NB chunks of TPC consecutive tokens (= CH = TPC*k consecutive assignments); NB is a
// few CTAs per SM so that the row copy of K2 fills the machine.
//   K1 perm_count   : CTA b histograms the slots of chunk b into hist[b][*].  The LAST CTA to
//                     finish (a ticket counter; no CTA ever waits for another) turns the
//                     table into per-slot exclusive prefixes over the chunks, and writes the
//                     slot totals and offsets[] (aligned exclusive scan of the totals).
//   K2 perm_scatter : CTA b ranks the assignments of chunk b IN ORDER (warp 0: match.any + a
//                     running counter per slot that starts at offsets[s] + hist[b][s]) => rows
//                     inside a slot are in ascending flat index (stable, bit-exact w.r.t. the
//                     counting-sort definition); writes assign_to_row / row_to_assign; then
//                     copies its TPC token rows: X[t,:] is read ONCE (16-byte vectors, the
//                     loads are issued before the ranking finishes) and stored to each of its
//                     <= k destination rows, so DRAM traffic is the algorithmic
//                     2*T_res*d + 2*R*d bytes.  Padding rows (align > 1) are zero-filled.
#include <atomic>

#include "common.cuh"

namespace vibe {
namespace {

constexpr int kMaxSlots = 1024;
constexpr int kMaxChunk = 1024;      // assignments per chunk (CH = TPC*k)
constexpr int kTargetChunks = 592;   // ~4 CTAs per SM
constexpr int kTickets = 64;

// Ticket counters of K1 (one per in-flight call, round-robin): zero at module load, and the
// last CTA of every call puts its counter back to zero.
__device__ unsigned int g_tickets[kTickets];

__device__ __forceinline__ int slot_of(const int32_t* __restrict__ ids, const int32_t* __restrict__ emap, int i,
                                       int E, int E_loc) {
  const int e = __ldg(ids + i);
  if (e < 0 || e >= E) return -1;
  const int s = emap ? __ldg(emap + e) : e;
  return (s >= 0 && s < E_loc) ? s : -1;
}

// K1 ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) perm_count_kernel(const int32_t* __restrict__ ids,
                                                          const int32_t* __restrict__ emap, int A, int E, int E_loc,
                                                          int CH, int NB, int align, int ticket,
                                                          int32_t* __restrict__ hist /*[NB][E_loc]*/,
                                                          int32_t* __restrict__ totals /*[E_loc]*/,
                                                          int32_t* __restrict__ offsets /*[E_loc+1]*/) {
  __shared__ int s_cnt[kMaxSlots];
  __shared__ int s_part[1024];
  __shared__ int s_last;
  const int tid = threadIdx.x;
  for (int s = tid; s < E_loc; s += 1024) s_cnt[s] = 0;
  __syncthreads();
  const int lo = blockIdx.x * CH, hi = min(A, lo + CH);
  for (int i = lo + tid; i < hi; i += 1024) {
    const int s = slot_of(ids, emap, i, E, E_loc);
    if (s >= 0) atomicAdd(&s_cnt[s], 1);
  }
  __syncthreads();
  int32_t* row = hist + (size_t)blockIdx.x * E_loc;
  for (int s = tid; s < E_loc; s += 1024) row[s] = s_cnt[s];
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(&g_tickets[ticket], 1u) == (unsigned)(NB - 1));
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (tid == 0) g_tickets[ticket] = 0;

  // ---- last CTA: hist[b][s] <- sum_{b' < b} hist[b'][s]; totals; offsets ----
  // Threads form G groups of W = min(E_loc, 1024) slot columns; group g owns the chunk rows
  // [g*RPG, (g+1)*RPG).  Pass 1: group sums; exclusive scan over the groups; pass 2: rewrite.
  for (int s0 = 0; s0 < E_loc; s0 += 1024) {
    const int W = min(E_loc - s0, 1024);
    const int G = 1024 / W;
    const int g = tid / W, c = tid - g * W;
    const bool act = g < G;
    const int RPG = (NB + G - 1) / G;
    const int b0 = min(NB, g * RPG), b1 = min(NB, b0 + RPG);
    volatile int32_t* col = hist + s0 + c;
    int sum = 0;
    if (act)
      for (int b = b0; b < b1; ++b) sum += col[(size_t)b * E_loc];
    s_part[tid] = act ? sum : 0;
    __syncthreads();
    int base = 0;
    if (act)
      for (int gg = 0; gg < g; ++gg) base += s_part[gg * W + c];
    if (act && g == G - 1) s_cnt[s0 + c] = base + sum;     // slot total
    if (act) {
      int run = base;
      for (int b = b0; b < b1; ++b) {
        const int v = col[(size_t)b * E_loc];
        col[(size_t)b * E_loc] = run;
        run += v;
      }
    }
    __syncthreads();
  }
  // offsets = exclusive scan of roundup(total, align) over <= 1024 slots (one value per thread)
  {
    const int lane = tid & 31, warp = tid >> 5;
    const int tot = (tid < E_loc) ? s_cnt[tid] : 0;
    const int v = ((tot + align - 1) / align) * align;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    __syncthreads();
    if (lane == 31) s_part[warp] = inc;
    __syncthreads();
    int woff = 0;
    for (int w = 0; w < warp; ++w) woff += s_part[w];
    if (tid < E_loc) {
      totals[tid] = tot;
      offsets[tid] = woff + inc - v;
      if (tid == E_loc - 1) offsets[E_loc] = woff + inc;
    }
  }
}

// K2 ------------------------------------------------------------------------------------
template <int UNROLL>
__global__ void __launch_bounds__(256) perm_scatter_kernel(const __nv_bfloat16* __restrict__ X,
                                                           const int32_t* __restrict__ ids,
                                                           const int32_t* __restrict__ emap, int T, int k, int d,
                                                           int E, int E_loc, int TPC, int align,
                                                           const int32_t* __restrict__ hist,
                                                           const int32_t* __restrict__ totals,
                                                           const int32_t* __restrict__ offsets,
                                                           int32_t* __restrict__ row_to_assign,
                                                           int32_t* __restrict__ assign_to_row,
                                                           __nv_bfloat16* __restrict__ Xp) {
  __shared__ int s_run[kMaxSlots];     // next row of every slot for this chunk
  __shared__ int s_dest[kMaxChunk];    // slot, then destination row, of every assignment of the chunk
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int b = blockIdx.x;
  const int t0 = b * TPC, t1 = min(T, t0 + TPC);
  const int lo = t0 * k, n_asg = (t1 - t0) * k;
  const int vpr = d >> 3;

  for (int i = tid; i < n_asg; i += 256) s_dest[i] = slot_of(ids, emap, lo + i, E, E_loc);
  for (int s = tid; s < E_loc; s += 256) s_run[s] = __ldg(offsets + s) + __ldg(hist + (size_t)b * E_loc + s);
  __syncthreads();

  // ---- first batch of row loads is in flight while warp 0 ranks ----
  const int n_vec = (t1 - t0) * vpr;     // 16-byte vectors of this chunk's token rows
  uint4 val[UNROLL];
  const uint4* src0 = reinterpret_cast<const uint4*>(X + (size_t)t0 * d);
  bool need[UNROLL];
#pragma unroll
  for (int q = 0; q < UNROLL; ++q) {
    const int v = tid + q * 256;
    need[q] = false;
    if (v < n_vec) {
      const int tt = v / vpr;
      for (int j = 0; j < k; ++j) need[q] |= (s_dest[tt * k + j] >= 0);
      if (need[q]) val[q] = ld_nc_v4(src0 + v);
    }
  }
  __syncthreads();   // every thread has read the slots it needs before warp 0 overwrites them

  if (warp == 0) {
    for (int i0 = 0; i0 < n_asg; i0 += 32) {
      const int i = i0 + lane;
      const int s = (i < n_asg) ? s_dest[i] : -1;
      const unsigned peers = __match_any_sync(0xffffffffu, s);
      int r = -1;
      if (s >= 0) r = s_run[s] + __popc(peers & ((1u << lane) - 1u));
      __syncwarp();
      if (s >= 0 && (peers >> lane) == 1u) s_run[s] += __popc(peers);   // highest peer lane updates
      __syncwarp();
      if (i < n_asg) {
        s_dest[i] = r;
        assign_to_row[lo + i] = r;
        if (r >= 0) row_to_assign[r] = lo + i;
      }
    }
  }
  __syncthreads();

  // ---- copy rows: vector v of the chunk = (token v / vpr, vector v % vpr) ----
  uint4* dst0 = reinterpret_cast<uint4*>(Xp);
  for (int vb = 0; vb < n_vec; vb += 256 * UNROLL) {
    if (vb > 0) {
#pragma unroll
      for (int q = 0; q < UNROLL; ++q) {
        const int v = vb + tid + q * 256;
        need[q] = false;
        if (v < n_vec) {
          const int tt = v / vpr;
          for (int j = 0; j < k; ++j) need[q] |= (s_dest[tt * k + j] >= 0);
          if (need[q]) val[q] = ld_nc_v4(src0 + v);
        }
      }
    }
#pragma unroll
    for (int q = 0; q < UNROLL; ++q) {
      const int v = vb + tid + q * 256;
      if (v < n_vec && need[q]) {
        const int tt = v / vpr;
        const int vv = v - tt * vpr;
        for (int j = 0; j < k; ++j) {
          const int r = s_dest[tt * k + j];
          if (r >= 0) st_na_v4(dst0 + (size_t)r * vpr + vv, val[q]);
        }
      }
    }
  }

  // ---- padding rows (align > 1): index -1, zero activations ----
  if (align > 1) {
    for (int s = b; s < E_loc; s += gridDim.x) {
      const int p0 = __ldg(offsets + s) + __ldg(totals + s), p1 = __ldg(offsets + s + 1);
      for (int r = p0 + warp; r < p1; r += 8) {
        if (lane == 0) row_to_assign[r] = -1;
        uint4* dst = dst0 + (size_t)r * vpr;
        for (int v = lane; v < vpr; v += 32) dst[v] = make_uint4(0, 0, 0, 0);
      }
    }
  }
}

struct Chunking {
  int TPC, CH, NB;
};
Chunking chunking(int T, int k) {
  Chunking c;
  int tpc = (T + kTargetChunks - 1) / kTargetChunks;
  if (tpc < 1) tpc = 1;
  const int max_tpc = kMaxChunk / k > 0 ? kMaxChunk / k : 1;
  if (tpc > max_tpc) tpc = max_tpc;
  c.TPC = tpc;
  c.CH = tpc * k;
  c.NB = T > 0 ? (T + tpc - 1) / tpc : 1;
  return c;
}

}  // namespace

size_t permute_ws_bytes(int T, int k, int E_loc) {
  const Chunking c = chunking(T, k);
  return round_up((size_t)c.NB * E_loc * sizeof(int32_t), 256) + round_up((size_t)E_loc * sizeof(int32_t), 256);
}

}  // namespace vibe

extern "C" int64_t vibe_rows_cap(int32_t T, int32_t k, int32_t E_loc, int32_t align) {
  if (T < 0 || k < 1 || E_loc < 1 || align < 1) return -1;
  const int64_t per_tok = k < E_loc ? k : E_loc;
  return (int64_t)T * per_tok + (int64_t)E_loc * (align - 1);
}

extern "C" vibe_status vibe_permute(const void* X, const int32_t* topk_ids, const int32_t* counts,
                                    const int32_t* expert_map, int32_t T, int32_t d, int32_t k, int32_t E,
                                    int32_t E_loc, int32_t align, void* Xp, int32_t* offsets,
                                    int32_t* row_to_assign, int32_t* assign_to_row, void* ws, size_t ws_bytes,
                                    void* stream) {
  using namespace vibe;
  (void)counts;  // advisory: the stable ranking needs per-chunk histograms anyway
  clear_error();
  VIBE_REQUIRE(T >= 0 && k >= 1 && E >= 1 && E_loc >= 1 && d >= 8, VIBE_ERR_INVALID_ARG,
               "vibe_permute: bad sizes T=%d k=%d E=%d E_loc=%d d=%d", T, k, E, E_loc, d);
  VIBE_REQUIRE(d % 8 == 0, VIBE_ERR_INVALID_ARG, "vibe_permute: d %% 8 != 0 (rows must be 16-byte multiples)");
  VIBE_REQUIRE(align >= 1, VIBE_ERR_INVALID_ARG, "vibe_permute: align < 1");
  VIBE_REQUIRE(k <= E, VIBE_ERR_INVALID_ARG, "vibe_permute: k > E");
  VIBE_REQUIRE(k <= kMaxChunk, VIBE_ERR_UNSUPPORTED, "vibe_permute: k > %d not implemented", kMaxChunk);
  VIBE_REQUIRE(E_loc <= E, VIBE_ERR_INVALID_ARG, "vibe_permute: E_loc > E");
  VIBE_REQUIRE(expert_map != nullptr || E_loc == E, VIBE_ERR_INVALID_ARG,
               "vibe_permute: expert_map NULL requires E_loc == E");
  VIBE_REQUIRE((int64_t)T * k < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "vibe_permute: T*k >= 2^31");
  VIBE_REQUIRE(vibe_rows_cap(T, k, E_loc, align) < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG,
               "vibe_permute: row capacity >= 2^31");
  VIBE_REQUIRE(E_loc <= kMaxSlots, VIBE_ERR_UNSUPPORTED, "vibe_permute: E_loc > %d not implemented", kMaxSlots);
  VIBE_REQUIRE(offsets != nullptr, VIBE_ERR_INVALID_ARG, "vibe_permute: offsets is NULL");
  VIBE_REQUIRE(T == 0 || (X && topk_ids && Xp && row_to_assign && assign_to_row), VIBE_ERR_INVALID_ARG,
               "vibe_permute: NULL tensor");
  VIBE_REQUIRE(T == 0 || (aligned16(X) && aligned16(Xp)), VIBE_ERR_INVALID_ARG,
               "vibe_permute: X / Xp must be 16-byte aligned");
  const size_t need = permute_ws_bytes(T, k, E_loc);
  VIBE_REQUIRE(ws != nullptr && ws_bytes >= need && aligned16(ws), VIBE_ERR_WORKSPACE,
               "vibe_permute: workspace needs %zu bytes, 16-byte aligned (got %zu)", need, ws_bytes);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int A = T * k;
  if (A == 0) {
    VIBE_CUDA(cudaMemsetAsync(offsets, 0, (size_t)(E_loc + 1) * sizeof(int32_t), st));
    return VIBE_OK;
  }
  const Chunking c = chunking(T, k);
  int32_t* hist = reinterpret_cast<int32_t*>(ws);
  int32_t* totals = reinterpret_cast<int32_t*>(reinterpret_cast<char*>(ws) +
                                               round_up((size_t)c.NB * E_loc * sizeof(int32_t), 256));
  static std::atomic<unsigned> next_ticket{0};
  const int ticket = (int)(next_ticket.fetch_add(1, std::memory_order_relaxed) % kTickets);
  perm_count_kernel<<<c.NB, 1024, 0, st>>>(topk_ids, expert_map, A, E, E_loc, c.CH, c.NB, align, ticket, hist, totals,
                                           offsets);
  VIBE_LAUNCH_CHECK("perm_count_kernel");
  perm_scatter_kernel<4><<<c.NB, 256, 0, st>>>(reinterpret_cast<const __nv_bfloat16*>(X), topk_ids, expert_map, T, k,
                                               d, E, E_loc, c.TPC, align, hist, totals, offsets, row_to_assign,
                                               assign_to_row, reinterpret_cast<__nv_bfloat16*>(Xp));
  VIBE_LAUNCH_CHECK("perm_scatter_kernel");
  return VIBE_OK;
}
