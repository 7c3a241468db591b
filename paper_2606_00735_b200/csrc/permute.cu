// permute.cu -- a3: stable counting sort of assignments by local expert slot + row gather
// (vibe_permute).  Semantics: include/vibe.h, readings P1-P4.
//
// Four small launches on one stream, no host sync, no spin-waits between CTAs:
//   K1 perm_hist     : every warp owns a contiguous chunk of kChunk assignments and writes
//                      its per-slot histogram (slot-major layout [E_loc][NW]).
//   K2 perm_scan     : one CTA per slot: exclusive scan over the NW chunk counts (in place)
//                      and the slot total.
//   K3 perm_index    : every CTA rebuilds offsets[] from the totals (<= 1024 slots, a block
//                      scan), every warp re-walks its chunk IN ORDER and ranks each
//                      assignment with match.any + a per-warp running counter in shared
//                      memory => rows inside a slot are in ascending flat index (stable,
//                      bit-exact w.r.t. the counting-sort definition).  Writes
//                      assign_to_row / row_to_assign; zero-fills padding rows.
//   K4 perm_rows     : token-major gather/scatter of the bf16 rows, one thread per 16-byte vector:
//                      X[t,:] is read ONCE and written to each of its <= k destination rows,
//                      so DRAM traffic equals the algorithmic 2*T_res*d + 2*R*d bytes.
//                      (E_loc < E: the row-major variant perm_rows_by_row, work ~ R.)
#include "common.cuh"

namespace vibe {
namespace {

constexpr int kChunk = 256;          // assignments per warp
constexpr int kWarpsPerBlock = 8;    // K1/K3 block = 256 threads
constexpr int kMaxSlots = 1024;

__device__ __forceinline__ int slot_of(const int32_t* __restrict__ ids, const int32_t* __restrict__ emap, int i,
                                       int E, int E_loc) {
  const int e = ids[i];
  if (e < 0 || e >= E) return -1;
  const int s = emap ? emap[e] : e;
  return (s >= 0 && s < E_loc) ? s : -1;
}

// K1 ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) perm_hist_kernel(const int32_t* __restrict__ ids,
                                                        const int32_t* __restrict__ emap, int A, int E, int E_loc,
                                                        int NW, int32_t* __restrict__ hist /*[E_loc][NW]*/) {
  extern __shared__ int s_cnt[];  // [kWarpsPerBlock][E_loc]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int c = blockIdx.x * kWarpsPerBlock + warp;
  int* cnt = s_cnt + warp * E_loc;
  for (int s = lane; s < E_loc; s += 32) cnt[s] = 0;
  __syncwarp();
  if (c < NW) {
    const int lo = c * kChunk, hi = min(A, lo + kChunk);
    for (int i = lo + lane; i < hi; i += 32) {
      const int s = slot_of(ids, emap, i, E, E_loc);
      if (s >= 0) atomicAdd(&cnt[s], 1);
    }
    __syncwarp();
    for (int s = lane; s < E_loc; s += 32) hist[(size_t)s * NW + c] = cnt[s];
  }
}

// K2 ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) perm_scan_kernel(int32_t* __restrict__ hist, int NW,
                                                        int32_t* __restrict__ totals /*[E_loc]*/) {
  __shared__ int s_warp[8];
  __shared__ int s_carry;
  int32_t* h = hist + (size_t)blockIdx.x * NW;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int base = 0; base < NW; base += 256) {
    const int i = base + threadIdx.x;
    const int v = (i < NW) ? h[i] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    int woff = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) woff += (w < warp) ? s_warp[w] : 0;
    const int carry = s_carry;
    if (i < NW) h[i] = carry + woff + inc - v;  // exclusive
    __syncthreads();
    if (threadIdx.x == 255) s_carry = carry + woff + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) totals[blockIdx.x] = s_carry;
}

// K3 ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) perm_index_kernel(const int32_t* __restrict__ ids,
                                                         const int32_t* __restrict__ emap, int A, int E, int E_loc,
                                                         int NW, int align, int d,
                                                         const int32_t* __restrict__ hist /*exclusive, [E_loc][NW]*/,
                                                         const int32_t* __restrict__ totals,
                                                         int32_t* __restrict__ offsets /*[E_loc+1]*/,
                                                         int32_t* __restrict__ row_to_assign,
                                                         int32_t* __restrict__ assign_to_row,
                                                         __nv_bfloat16* __restrict__ Xp) {
  extern __shared__ int s_mem[];
  int* s_off = s_mem;                   // [E_loc+1] aligned segment starts
  int* s_run = s_mem + (E_loc + 1);     // [kWarpsPerBlock][E_loc] running base per warp
  __shared__ int s_warp[8];
  __shared__ int s_carry;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // ---- offsets = exclusive scan of roundup(total, align) (every CTA, redundantly) ----
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int base = 0; base < E_loc; base += 256) {
    const int i = base + threadIdx.x;
    const int v = (i < E_loc) ? ((totals[i] + align - 1) / align) * align : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    int woff = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) woff += (w < warp) ? s_warp[w] : 0;
    const int carry = s_carry;
    if (i < E_loc) s_off[i] = carry + woff + inc - v;
    __syncthreads();
    if (threadIdx.x == 255) s_carry = carry + woff + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) s_off[E_loc] = s_carry;
  __syncthreads();
  if (blockIdx.x == 0)
    for (int i = threadIdx.x; i <= E_loc; i += 256) offsets[i] = s_off[i];

  // ---- stable ranks for this warp's chunk ----
  const int c = blockIdx.x * kWarpsPerBlock + warp;
  int* run = s_run + warp * E_loc;
  if (c < NW) {
    for (int s = lane; s < E_loc; s += 32) run[s] = s_off[s] + hist[(size_t)s * NW + c];
    __syncwarp();
    const int lo = c * kChunk, hi = min(A, lo + kChunk);
    for (int i0 = lo; i0 < hi; i0 += 32) {
      const int i = i0 + lane;
      const int s = (i < hi) ? slot_of(ids, emap, i, E, E_loc) : -1;
      const unsigned peers = __match_any_sync(0xffffffffu, s);
      int r = -1;
      if (s >= 0) {
        const unsigned lt = peers & ((1u << lane) - 1u);
        r = run[s] + __popc(lt);
      }
      __syncwarp();
      if (s >= 0 && (peers >> lane) == 1u) run[s] += __popc(peers);  // highest peer lane updates
      __syncwarp();
      if (i < hi) {
        assign_to_row[i] = r;
        if (r >= 0) row_to_assign[r] = i;
      }
    }
  }
  // ---- padding rows (align > 1): index -1, zero activations ----
  if (align > 1) {
    const int vec_per_row = d / 8;
    for (int s = blockIdx.x; s < E_loc; s += gridDim.x) {
      const int p0 = s_off[s] + totals[s], p1 = s_off[s + 1];
      for (int r = p0 + warp; r < p1; r += kWarpsPerBlock) {
        if (lane == 0) row_to_assign[r] = -1;
        uint4* dst = reinterpret_cast<uint4*>(Xp + (size_t)r * d);
        for (int v = lane; v < vec_per_row; v += 32) dst[v] = make_uint4(0, 0, 0, 0);
      }
    }
  }
}

// K4 ------------------------------------------------------------------------------------
// One thread per VPT 16-byte vectors of one token row (vectors v and v + vpr/2 when VPT == 2):
// the vector is read once and stored to each of the token's <= k destination rows.  The k
// row indices are warp-uniform addresses (one broadcast transaction, L1-resident).  No
// grid-stride loop: the grid covers T * vpr / VPT threads.
template <int VPT>
__global__ void __launch_bounds__(256) perm_rows_kernel(const __nv_bfloat16* __restrict__ X,
                                                        const int32_t* __restrict__ assign_to_row, int T, int k,
                                                        int d, __nv_bfloat16* __restrict__ Xp) {
  const int vpr = d >> 3;
  const int per_row = vpr / VPT;
  const long long g = (long long)blockIdx.x * 256 + threadIdx.x;
  if (g >= (long long)T * per_row) return;
  const int t = (int)(g / per_row);
  const int v0 = (int)(g - (long long)t * per_row);
  const int32_t* a2r = assign_to_row + (size_t)t * k;
  bool any = false;
  for (int j = 0; j < k; ++j) any |= (__ldg(a2r + j) >= 0);
  if (!any) return;
  const uint4* src = reinterpret_cast<const uint4*>(X + (size_t)t * d) + v0;
  uint4 val[VPT];
#pragma unroll
  for (int q = 0; q < VPT; ++q) val[q] = ld_nc_v4(src + q * per_row);
  for (int j = 0; j < k; ++j) {
    const int r = __ldg(a2r + j);
    if (r < 0) continue;
    uint4* dst = reinterpret_cast<uint4*>(Xp + (size_t)r * d) + v0;
#pragma unroll
    for (int q = 0; q < VPT; ++q) st_na_v4(dst + q * per_row, val[q]);
  }
}

// K4' -----------------------------------------------------------------------------------
// Row-major variant for expert-parallel shards (E_loc < E), where only a fraction of the
// T*k assignments is resident: persistent warps walk the R = offsets[E_loc] real rows
// (extent read on the device) and copy X[row_to_assign[r] / k, :] -> Xp[r, :], UNROLL
// independent 16-byte loads in flight per lane.  Work is proportional to R, not to T*k.
template <int UNROLL>
__global__ void __launch_bounds__(256) perm_rows_by_row_kernel(const __nv_bfloat16* __restrict__ X,
                                                               const int32_t* __restrict__ row_to_assign,
                                                               const int32_t* __restrict__ offsets, int E_loc,
                                                               int k, int d, __nv_bfloat16* __restrict__ Xp) {
  const int R = __ldg(offsets + E_loc);
  const int lane = threadIdx.x & 31;
  const int nwarps = gridDim.x * (256 / 32);
  const int vpr = d >> 3;
  for (int r = blockIdx.x * (256 / 32) + (threadIdx.x >> 5); r < R; r += nwarps) {
    const int i = __ldg(row_to_assign + r);
    if (i < 0) continue;   // padding row: already zero-filled by perm_index_kernel
    const uint4* src = reinterpret_cast<const uint4*>(X + (size_t)(i / k) * d);
    uint4* dst = reinterpret_cast<uint4*>(Xp + (size_t)r * d);
    for (int v0 = lane; v0 < vpr; v0 += 32 * UNROLL) {
      uint4 val[UNROLL];
#pragma unroll
      for (int q = 0; q < UNROLL; ++q)
        if (v0 + 32 * q < vpr) val[q] = ld_nc_v4(src + v0 + 32 * q);
#pragma unroll
      for (int q = 0; q < UNROLL; ++q)
        if (v0 + 32 * q < vpr) st_na_v4(dst + v0 + 32 * q, val[q]);
    }
  }
}

}  // namespace

size_t permute_ws_bytes(int T, int k, int E_loc) {
  const int64_t A = (int64_t)T * k;
  const int64_t NW = (A + kChunk - 1) / kChunk;
  return round_up((size_t)(NW > 0 ? NW : 1) * E_loc * sizeof(int32_t), 256) +
         round_up((size_t)E_loc * sizeof(int32_t), 256);
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
  const int NW = (A + kChunk - 1) / kChunk;
  int32_t* hist = reinterpret_cast<int32_t*>(ws);
  int32_t* totals = reinterpret_cast<int32_t*>(reinterpret_cast<char*>(ws) +
                                               round_up((size_t)NW * E_loc * sizeof(int32_t), 256));
  const int nblk = (NW + kWarpsPerBlock - 1) / kWarpsPerBlock;
  const size_t smem1 = (size_t)kWarpsPerBlock * E_loc * sizeof(int);
  const size_t smem3 = (size_t)(E_loc + 1 + kWarpsPerBlock * E_loc) * sizeof(int);
  perm_hist_kernel<<<nblk, 256, smem1, st>>>(topk_ids, expert_map, A, E, E_loc, NW, hist);
  VIBE_LAUNCH_CHECK("perm_hist_kernel");
  perm_scan_kernel<<<E_loc, 256, 0, st>>>(hist, NW, totals);
  VIBE_LAUNCH_CHECK("perm_scan_kernel");
  perm_index_kernel<<<nblk, 256, smem3, st>>>(topk_ids, expert_map, A, E, E_loc, NW, align, d, hist, totals, offsets,
                                              row_to_assign, assign_to_row, reinterpret_cast<__nv_bfloat16*>(Xp));
  VIBE_LAUNCH_CHECK("perm_index_kernel");
  const int vpr = d / 8;
  const __nv_bfloat16* Xb = reinterpret_cast<const __nv_bfloat16*>(X);
  __nv_bfloat16* Xpb = reinterpret_cast<__nv_bfloat16*>(Xp);
  if (E_loc < E) {
    // expert-parallel shard: work proportional to the resident rows
    perm_rows_by_row_kernel<4><<<num_sms() * 8, 256, 0, st>>>(Xb, row_to_assign, offsets, E_loc, k, d, Xpb);
  } else {
    const int vpt = (vpr % 2 == 0) ? 2 : 1;
    const long long blocks = ((long long)T * (vpr / vpt) + 255) / 256;
    VIBE_REQUIRE(blocks < (1ll << 31), VIBE_ERR_UNSUPPORTED, "vibe_permute: T*d too large for one launch");
    if (vpt == 2)
      perm_rows_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(Xb, assign_to_row, T, k, d, Xpb);
    else
      perm_rows_kernel<1><<<(unsigned)blocks, 256, 0, st>>>(Xb, assign_to_row, T, k, d, Xpb);
  }
  VIBE_LAUNCH_CHECK("perm_rows_kernel");
  return VIBE_OK;
}
