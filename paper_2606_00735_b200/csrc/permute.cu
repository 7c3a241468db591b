// permute.cu -- a3: stable counting sort of assignments by local expert slot + row gather
// (vibe_permute).  Semantics: include/vibe.h, readings P1-P4.
//
// Two launches on one stream, no host sync:
//   K1 perm_index  : a COOPERATIVE launch of G <= #SMs CTAs x 1024 threads (all co-resident, so
//                    the one grid-wide barrier below cannot deadlock); when G <= 8 the grid is one
//                    thread-block cluster instead and the barrier is barrier.cluster.  Warp gw = 32*cta + w owns
//                    the contiguous chunk [gw*WCH, (gw+1)*WCH) of the A = T*k assignments.
//                      pass 1  lanes holding the same slot are matched with ballots (one per key
//                              bit, fixed cost); per-warp slot histograms in shared memory; the
//                              matching (lanes below me, group size, leader) is parked in
//                              assign_to_row so that pass 2 needs no votes
//                      scan    exclusive prefix over the 32 warps of the CTA per slot; the CTA
//                              totals go to a [G][E_loc] table in the workspace; GRID BARRIER;
//                              every CTA sums the rows of the CTAs before it (its base) and all
//                              rows (slot totals), and derives offsets[] (aligned exclusive scan)
//                      pass 2  every warp re-walks its chunk IN ORDER: row = base + running
//                              counter + lanes below me => rows inside a slot are in ascending
//                              flat index (stable, bit-exact w.r.t. the counting-sort
//                              definition).  Writes assign_to_row / row_to_assign; zero-fills
//                              padding rows (align > 1).
//                    (A single 8-CTA cluster with a DSMEM exchange was measured first: 8 SMs are
//                    too few -- the scattered 4-byte row_to_assign stores and the votes of 256
//                    warps saturate their LSU/vote pipes: 17 us at A = 64K, 105 us at A = 512K.)
//   K2 perm_rows   : token-major gather/scatter of the bf16 rows, one thread per 16-byte vector:
//                    X[t,:] is read ONCE and written to each of its <= k destination rows,
//                    so DRAM traffic equals the algorithmic 2*T_res*d + 2*R*d bytes.
//                    (E_loc < E: the row-major variant perm_rows_by_row, work ~ R.)
#include <atomic>
#include <mutex>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

constexpr int kMaxSlots = 1024;
constexpr int kIdxThreads = 1024;
constexpr int kIdxWarps = kIdxThreads / 32;
constexpr int kBatch = 8;            // id loads in flight per lane
static_assert(kIdxWarps == 32, "the offsets scan keeps one warp partial per lane");

// Grid-barrier state of K1: two counters {arrived, departed} at the end of the CALLER's workspace, zeroed by a
// memset node in front of the launch -- calls that may run concurrently (other streams, replayed graphs) must
// not share a workspace anyway (the table of CTA totals lives there), so they never share a barrier either.

__device__ __forceinline__ int slot_of(const int32_t* __restrict__ ids, const int32_t* __restrict__ emap, int i,
                                       int E, int E_loc) {
  const int e = __ldg(ids + i);
  if (e < 0 || e >= E) return -1;
  const int s = emap ? __ldg(emap + e) : e;
  return (s >= 0 && s < E_loc) ? s : -1;
}

// Lanes of the warp that hold the same key (key in [0, 2^nbits)): nbits ballots, fixed cost.
__device__ __forceinline__ unsigned same_key_lanes(int key, int nbits) {
  unsigned peers = 0xffffffffu;
  for (int b = 0; b < nbits; ++b) {
    const bool bit = (key >> b) & 1;
    const unsigned bal = __ballot_sync(0xffffffffu, bit);
    peers &= bit ? bal : ~bal;
  }
  return peers;
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// All G CTAs of the (cooperative) grid meet here once.
__device__ __forceinline__ void grid_barrier_once(unsigned* bar, unsigned G) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(&bar[0], 1u);
    while (ld_acquire_u32(&bar[0]) < G) __nanosleep(32);
    __threadfence();
    atomicAdd(&bar[1], 1u);                  // (kept for debugging: departed == G when the kernel ends)
  }
  __syncthreads();
}

// K1 ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kIdxThreads, 1)
perm_index_kernel(const int32_t* __restrict__ ids, const int32_t* __restrict__ emap, int A, int E, int E_loc,
                  int WCH, int align, int d, unsigned int* bar /* NULL: the grid is ONE cluster */,
                  int32_t* __restrict__ tbl /*[G][E_loc]*/,
                  int32_t* __restrict__ offsets /*[E_loc+1]*/, int32_t* __restrict__ row_to_assign,
                  int32_t* __restrict__ assign_to_row, __nv_bfloat16* __restrict__ Xp) {
  extern __shared__ int s_mem[];
  int* s_wh = s_mem;                            // [kIdxWarps][E_loc] per-warp counts -> running row
  int* s_base = s_wh + kIdxWarps * E_loc;       // [E_loc] offsets[s] + rows of the preceding CTAs
  int* s_tot = s_base + E_loc;                  // [E_loc] slot totals of the whole batch
  int* s_off = s_tot + E_loc;                   // [E_loc+1] aligned segment starts
  int* s_red = s_off + E_loc + 1;               // [2][kIdxThreads] partial sums of the table walk
  __shared__ int s_scan[kIdxWarps];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cta = blockIdx.x, G = gridDim.x;
  const int gw = cta * kIdxWarps + warp;
  const int lo = min(A, gw * WCH), hi = min(A, lo + WCH);
  int* wh = s_wh + warp * E_loc;
  const int nbits = 32 - __clz(E_loc);   // keys are slot + 1 in [0, E_loc]

  // programmatic dependent launch: K2's CTAs may become resident now; they wait in
  // griddepcontrol.wait until this grid has completed and flushed
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  for (int s = lane; s < E_loc; s += 32) wh[s] = 0;
  __syncwarp();
  // ---- pass 1 (kBatch independent id loads are in flight before the first one is consumed) ----
  for (int i0 = lo; i0 < hi; i0 += 32 * kBatch) {
    int sl[kBatch];
#pragma unroll
    for (int q = 0; q < kBatch; ++q) {
      const int i = i0 + q * 32 + lane;
      sl[q] = (i < hi) ? slot_of(ids, emap, i, E, E_loc) : -1;
    }
#pragma unroll
    for (int q = 0; q < kBatch; ++q) {
      if (i0 + q * 32 >= hi) break;           // warp-uniform
      const int i = i0 + q * 32 + lane;
      const int s = sl[q];
      const unsigned peers = same_key_lanes(s + 1, nbits);
      const int below = __popc(peers & ((1u << lane) - 1u));
      const int size = __popc(peers);
      const bool leader = (peers >> lane) == 1u;           // highest lane of the group
      if (s >= 0 && leader) wh[s] += size;
      if (i < hi) assign_to_row[i] = (s >= 0) ? (below | (size << 6) | ((int)leader << 12)) : -1;
      __syncwarp();
    }
  }
  __syncthreads();
  // ---- exclusive prefix over the warps of this CTA, per slot; CTA totals -> table ----
  for (int s = tid; s < E_loc; s += kIdxThreads) {
    int run = 0;
#pragma unroll 8
    for (int w = 0; w < kIdxWarps; ++w) {
      const int v = s_wh[w * E_loc + s];
      s_wh[w * E_loc + s] = run;
      run += v;
    }
    tbl[(size_t)cta * E_loc + s] = run;
  }
  if (bar == nullptr) {
    __threadfence();
    ptx::cluster_sync_all();          // G <= 8: hardware cluster barrier (release / acquire at cluster scope)
  } else {
    grid_barrier_once(bar, (unsigned)G);
  }
  // ---- walk the table: rows before mine (base) and all rows (totals).  W slot columns x
  // NG row groups; group g takes rows g, g + NG, ... ----
  for (int s0 = 0; s0 < E_loc; s0 += kIdxThreads) {
    const int W = min(E_loc - s0, kIdxThreads);
    // (row groups beyond G would have no row; the sums below run over NG: 128 -> 8 terms at 8 slots and 8 CTAs, 0.8 us)
    const int NG = min(kIdxThreads / W, G);
    const int g = tid / W, c = tid - g * W;
    int pre = 0, total = 0;
    if (g < NG) {
      const int32_t* col = tbl + s0 + c;
#pragma unroll 4
      for (int r = g; r < G; r += NG) {
        const int v = __ldcg(col + (size_t)r * E_loc);
        pre += (r < cta) ? v : 0;
        total += v;
      }
    }
    s_red[tid] = pre;
    s_red[kIdxThreads + tid] = total;
    __syncthreads();
    if (tid < W) {
      int p = 0, t = 0;
      for (int gg = 0; gg < NG; ++gg) {
        p += s_red[gg * W + tid];
        t += s_red[kIdxThreads + gg * W + tid];
      }
      s_base[s0 + tid] = p;
      s_tot[s0 + tid] = t;
    }
    __syncthreads();
  }
  // ---- offsets = exclusive scan of roundup(total, align) over <= 1024 slots (one per thread) ----
  {
    const int tot = (tid < E_loc) ? s_tot[tid] : 0;
    const int v = ((tot + align - 1) / align) * align;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) s_scan[warp] = inc;
    __syncthreads();
    int part = s_scan[lane];                 // kIdxWarps == 32: one partial per lane
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, part, o);
      if (lane >= o) part += n;
    }
    const int woff = __shfl_sync(0xffffffffu, part, (warp + 31) & 31) * (warp > 0);
    if (tid < E_loc) {
      const int start = woff + inc - v;
      s_off[tid] = start;
      s_base[tid] += start;
      if (tid == E_loc - 1) s_off[E_loc] = woff + inc;
    }
    __syncthreads();
    if (cta == 0)
      for (int i = tid; i <= E_loc; i += kIdxThreads) offsets[i] = s_off[i];
  }
  // ---- pass 2: stable ranks (no votes: the parked matching + the running counters) ----
  for (int i0 = lo; i0 < hi; i0 += 32 * kBatch) {
    int sl[kBatch], pk[kBatch];
#pragma unroll
    for (int q = 0; q < kBatch; ++q) {
      const int i = i0 + q * 32 + lane;
      sl[q] = (i < hi) ? slot_of(ids, emap, i, E, E_loc) : -1;
      pk[q] = (i < hi) ? assign_to_row[i] : -1;
    }
#pragma unroll
    for (int q = 0; q < kBatch; ++q) {
      if (i0 + q * 32 >= hi) break;           // warp-uniform
      const int i = i0 + q * 32 + lane;
      const int s = sl[q];
      int r = -1;
      if (s >= 0) r = s_base[s] + wh[s] + (pk[q] & 63);
      __syncwarp();
      if (s >= 0 && (pk[q] >> 12)) wh[s] += (pk[q] >> 6) & 63;
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
    for (int s = cta; s < E_loc; s += G) {
      const int p0 = s_off[s] + s_tot[s], p1 = s_off[s + 1];
      for (int r = p0 + warp; r < p1; r += kIdxWarps) {
        if (lane == 0) row_to_assign[r] = -1;
        uint4* dst = reinterpret_cast<uint4*>(Xp + (size_t)r * d);
        for (int v = lane; v < vec_per_row; v += 32) dst[v] = make_uint4(0, 0, 0, 0);
      }
    }
  }
}

// K2 ------------------------------------------------------------------------------------
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
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the FFN's CTAs may become resident
  const long long g = (long long)blockIdx.x * 256 + threadIdx.x;
  const bool live = g < (long long)T * per_row;
  const int t = live ? (int)(g / per_row) : 0;
  const int v0 = live ? (int)(g - (long long)t * per_row) : 0;
  // X is an INPUT of the permutation (not written by the index kernel): the CTAs that are resident while K1 still
  // runs issue their row loads before they wait for the index
  const uint4* src = reinterpret_cast<const uint4*>(X + (size_t)t * d) + v0;
  uint4 val[VPT];
#pragma unroll
  for (int q = 0; q < VPT; ++q) val[q] = live ? ld_nc_v4(src + q * per_row) : make_uint4(0, 0, 0, 0);
  asm volatile("griddepcontrol.wait;" ::: "memory");     // K1's index is complete and visible
  if (!live) return;
  const int32_t* a2r = assign_to_row + (size_t)t * k;
  for (int j = 0; j < k; ++j) {
    const int r = __ldg(a2r + j);
    if (r < 0) continue;
    uint4* dst = reinterpret_cast<uint4*>(Xp + (size_t)r * d) + v0;
#pragma unroll
    for (int q = 0; q < VPT; ++q) st_na_v4(dst + q * per_row, val[q]);
  }
}

// K2' -----------------------------------------------------------------------------------
// Row-major variant for expert-parallel shards (E_loc < E), where only a fraction of the
// T*k assignments is resident: persistent warps walk the R = offsets[E_loc] real rows
// (extent read on the device) and copy X[row_to_assign[r] / k, :] -> Xp[r, :], UNROLL
// independent 16-byte loads in flight per lane.  Work is proportional to R, not to T*k.
template <int UNROLL>
__global__ void __launch_bounds__(256) perm_rows_by_row_kernel(const __nv_bfloat16* __restrict__ X,
                                                               const int32_t* __restrict__ row_to_assign,
                                                               const int32_t* __restrict__ offsets, int E_loc,
                                                               int k, int d, __nv_bfloat16* __restrict__ Xp) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the FFN's CTAs may become resident
  asm volatile("griddepcontrol.wait;" ::: "memory");     // K1's index is complete and visible
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
  (void)T;
  (void)k;
  // [G][E_loc] table of CTA slot totals, G <= number of SMs, + the grid-barrier counters
  return round_up((size_t)num_sms() * E_loc * sizeof(int32_t), 256) + 256;
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
  // K1: G CTAs, all co-resident (cooperative launch); WCH assignments per warp, a multiple of 32
  int G = (A + kIdxThreads - 1) / kIdxThreads;
  if (G > num_sms()) G = num_sms();
  const int warps = G * kIdxWarps;
  int WCH = (((A + warps - 1) / warps) + 31) / 32 * 32;
  const size_t smem1 = (size_t)((kIdxWarps + 3) * E_loc + 1 + 2 * kIdxThreads) * sizeof(int);
  static std::atomic<size_t> smem_set[kMaxDevices];   // per device: the opt-in above 48 KB is a per-device attribute
  std::atomic<size_t>& set = smem_set[current_device()];
  if (smem1 > 48 * 1024 && smem1 > set.load()) {
    VIBE_CUDA(cudaFuncSetAttribute(perm_index_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem1));
    set.store(smem1);
  }
  __nv_bfloat16* Xpb = reinterpret_cast<__nv_bfloat16*>(Xp);
  int32_t* tbl = reinterpret_cast<int32_t*>(ws);
  if (G <= 8) {
    // small batches: the whole grid is one thread-block cluster (portable size <= 8), the barrier is
    // barrier.cluster -- ~3 us less than the cooperative launch + atomic barrier at A = 8K
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)G;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cudaLaunchConfig_t lc1 = {};
    lc1.gridDim = dim3(G);
    lc1.blockDim = dim3(kIdxThreads);
    lc1.dynamicSmemBytes = smem1;
    lc1.stream = st;
    lc1.attrs = at;
    lc1.numAttrs = 1;
    VIBE_CUDA(cudaLaunchKernelEx(&lc1, perm_index_kernel, topk_ids, expert_map, (int)A, (int)E, (int)E_loc, WCH,
                                 (int)align, (int)d, (unsigned int*)nullptr, tbl, offsets, row_to_assign,
                                 assign_to_row, Xpb));
  } else {
    unsigned int* bar = reinterpret_cast<unsigned int*>(reinterpret_cast<char*>(ws) +
                                                        round_up((size_t)num_sms() * E_loc * sizeof(int32_t), 256));
    VIBE_CUDA(cudaMemsetAsync(bar, 0, 2 * sizeof(unsigned int), st));
    int A_ = A, E_ = E, El_ = E_loc, al_ = align, d_ = d;
    void* args[] = {(void*)&topk_ids, (void*)&expert_map, &A_, &E_, &El_, &WCH, &al_, &d_, &bar, &tbl, &offsets,
                    &row_to_assign, &assign_to_row, &Xpb};
    VIBE_CUDA(cudaLaunchCooperativeKernel((const void*)perm_index_kernel, dim3(G), dim3(kIdxThreads), args, smem1,
                                          st));
  }
  count_launch();
  const int vpr = d / 8;
  const __nv_bfloat16* Xb = reinterpret_cast<const __nv_bfloat16*>(X);
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t lc = {};
  lc.blockDim = dim3(256);
  lc.dynamicSmemBytes = 0;
  lc.stream = st;
  lc.attrs = pdl;
  lc.numAttrs = 1;
  const int32_t* r2a_c = row_to_assign;
  const int32_t* a2r_c = assign_to_row;
  const int32_t* off_c = offsets;
  if (E_loc < E) {
    // expert-parallel shard: work proportional to the resident rows
    lc.gridDim = dim3(num_sms() * 8);
    VIBE_CUDA(cudaLaunchKernelEx(&lc, perm_rows_by_row_kernel<4>, Xb, r2a_c, off_c, (int)E_loc, (int)k, (int)d, Xpb));
  } else {
    const int vpt = (vpr % 2 == 0) ? 2 : 1;
    const long long blocks = ((long long)T * (vpr / vpt) + 255) / 256;
    VIBE_REQUIRE(blocks < (1ll << 31), VIBE_ERR_UNSUPPORTED, "vibe_permute: T*d too large for one launch");
    lc.gridDim = dim3((unsigned)blocks);
    if (vpt == 2)
      VIBE_CUDA(cudaLaunchKernelEx(&lc, perm_rows_kernel<2>, Xb, a2r_c, (int)T, (int)k, (int)d, Xpb));
    else
      VIBE_CUDA(cudaLaunchKernelEx(&lc, perm_rows_kernel<1>, Xb, a2r_c, (int)T, (int)k, (int)d, Xpb));
  }
  VIBE_LAUNCH_CHECK("perm_rows_kernel");
  return VIBE_OK;
}

// ------------------------------------------------------------------------------------------------------------
// vibe_permute_static: vibe_permute for callers that cannot allocate device memory (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  The index kernel's scratch -- the [CTAs][E_loc] table of
// slot totals and the grid-barrier counters -- lives in a file-scope device array of VIBE_PERMUTE_STATIC_BYTES
// (304 KiB: E_loc <= 512 on the 148 SMs of a B200); every GPU that loads the library holds it until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the device address is taken once per
// device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels get.
// All calls share the array: calls that overlap on the GPU (two streams, graphs replayed side by side) race on it.
// It keeps the last call's contents; what must start at zero -- the barrier counters of the cooperative path -- is
// cleared by every call (vibe_permute does that for any workspace), the table is written before it is read.
// No cudaMalloc / cudaFree / allocating library routine is called.
// ------------------------------------------------------------------------------------------------------------
namespace vibe {
namespace {
static __device__ __align__(256) unsigned char g_permute_static_scratch[VIBE_PERMUTE_STATIC_BYTES];

vibe_status permute_static_scratch(void** out) {
  static std::mutex mu;
  static void* ptr[kMaxDevices] = {};
  const int dev = current_device();
  std::lock_guard<std::mutex> lk(mu);
  if (ptr[dev] == nullptr) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_permute_static_scratch);
    VIBE_REQUIRE(e == cudaSuccess && p != nullptr, VIBE_ERR_CUDA,
                 "vibe_permute_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return VIBE_OK;
}
}  // namespace
}  // namespace vibe

extern "C" vibe_status vibe_permute_static(const void* X, const int32_t* topk_ids, const int32_t* counts,
                                           const int32_t* expert_map, int32_t T, int32_t d, int32_t k, int32_t E,
                                           int32_t E_loc, int32_t align, void* Xp, int32_t* offsets,
                                           int32_t* row_to_assign, int32_t* assign_to_row, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(T >= 0 && k >= 1 && E >= 1 && E_loc >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_permute_static: bad sizes T=%d k=%d E=%d E_loc=%d", T, k, E, E_loc);
  const size_t need = permute_ws_bytes(T, k, E_loc);
  VIBE_REQUIRE(need <= (size_t)VIBE_PERMUTE_STATIC_BYTES, VIBE_ERR_WORKSPACE,
               "vibe_permute_static: E_loc=%d on %d SMs needs %zu bytes of scratch, the static array holds %d "
               "(use vibe_permute with a caller-provided workspace)",
               E_loc, num_sms(), need, (int)VIBE_PERMUTE_STATIC_BYTES);
  void* scratch = nullptr;
  const vibe_status s = permute_static_scratch(&scratch);
  if (s != VIBE_OK) return s;
  return vibe_permute(X, topk_ids, counts, expert_map, T, d, k, E, E_loc, align, Xp, offsets, row_to_assign,
                      assign_to_row, scratch, (size_t)VIBE_PERMUTE_STATIC_BYTES, stream);
}
