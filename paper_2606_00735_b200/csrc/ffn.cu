// ffn.cu -- a4: grouped SwiGLU expert FFN (vibe_grouped_ffn) on 5th-gen tensor cores.
//
// Two launches of one persistent, warp-specialised tcgen05 kernel (one CTA per SM):
//   GEMM-1  H[r, n0:n0+128]  = silu(Xp[r,:] W1[s][:, n0:..]) * (Xp[r,:] W3[s][:, n0:..])   K = d
//           one UMMA of N = 256 per K-step: columns 0..127 gate, 128..255 up; SwiGLU is
//           applied in the epilogue straight out of TMEM (H never exists in fp32 in HBM).
//   GEMM-2  Y[r, n0:n0+256]  = H[r,:] W2[s][:, n0:..]                                     K = f
// Operands:
//   A (activations, K-major)   : ONE 2-D TMA map over all permuted rows; the row coordinate
//                                is offsets[s] + 128*m_blk, taken from the device-side
//                                offsets -> no per-expert descriptors, no host sync.
//   B (weights [E_loc,K,N], N contiguous = "MN-major") : ONE 3-D TMA map (N, K, E_loc),
//                                consumed IN PLACE through MN-major UMMA descriptors --
//                                no weight repacking.
// Rows of a 128-row tile that spill past the end of the expert's segment are computed and
// masked at the store; rows past R_cap are zero-filled by TMA.
// Pipeline: warp 0 = TMA producer, warp 1 = UMMA issuer (+ TMEM owner), warps 2..5 = epilogue.
// 4 smem stages x 48 KB (A 128x64, B 256x64), 2 TMEM accumulator stages x 256 columns so the
// epilogue of tile i overlaps the MMAs of tile i+1.
// Tile order: expert-major, then n-block, then m-block fastest, so CTAs that run at the
// same time share the same weight tile through L2 and each weight byte leaves HBM once.
//
// Semantics: include/vibe.h (vibe_grouped_ffn); F1-F4.
#include <mutex>
#include <unordered_map>
#include <string>
#include <cstring>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

constexpr int BM = 128;                 // rows per tile (UMMA M)
constexpr int BK = 64;                  // K per smem stage (one 128-byte swizzle atom of bf16)
constexpr int UMMA_N = 256;             // accumulator columns per tile
constexpr int UMMA_K = 16;
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 2;            // 16 KB
constexpr int B_ATOM_BYTES = 64 * BK * 2;       // 8 KB : 64 N-columns x 64 K-rows
constexpr int B_BYTES = 4 * B_ATOM_BYTES;       // 32 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 48 KB
constexpr int NUM_THREADS = 192;
constexpr int MAX_SLOTS = 1024;
constexpr int TMEM_COLS = 512;

struct SmemTail {
  uint64_t full[STAGES];
  uint64_t empty[STAGES];
  uint64_t tfull[2];
  uint64_t tempty[2];
  uint32_t tmem_base;
  int32_t total_m_tiles;
  int32_t off[MAX_SLOTS + 1];     // segment starts (rows)
  int32_t cum[MAX_SLOTS + 1];     // exclusive prefix of m-tiles per slot
};
constexpr size_t SMEM_BYTES = 1024 + (size_t)STAGES * STAGE_BYTES + sizeof(SmemTail);

struct TileCursor {
  int e = 0;
  // Decode tile id -> (slot e, m_blk, n_blk).  Tiles ids are monotone per CTA, so e only advances.
  __device__ __forceinline__ void decode(const SmemTail* t, int tile, int NB, int& m_blk, int& n_blk) {
    while (tile >= t->cum[e + 1] * NB) ++e;
    const int local = tile - t->cum[e] * NB;
    const int mt = t->cum[e + 1] - t->cum[e];
    n_blk = local / mt;
    m_blk = local - n_blk * mt;
  }
};

__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

template <bool kGateUp>
__global__ void __launch_bounds__(NUM_THREADS, 1)
ffn_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
                const __grid_constant__ CUtensorMap tmB1, const int32_t* __restrict__ offsets, int E_loc,
                int n_total, int k_total, __nv_bfloat16* __restrict__ out, int ld_out) {
  constexpr int BN_OUT = kGateUp ? 128 : 256;  // output columns per tile
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  SmemTail* tail = reinterpret_cast<SmemTail*>(smem + (size_t)STAGES * STAGE_BYTES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int NB = (n_total + BN_OUT - 1) / BN_OUT;
  const int KB = k_total / BK;

  // ------------------------------------------------------------------ setup
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tmA);
    ptx::prefetch_tensormap(&tmB0);
    if (kGateUp) ptx::prefetch_tensormap(&tmB1);
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(ptx::smem_u32(&tail->full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->empty[s]), 1);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(ptx::smem_u32(&tail->tfull[a]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->tempty[a]), 4);
    }
    ptx::fence_barrier_init();
  } else if (warp == 1) {
    ptx::tmem_alloc(ptx::smem_u32(&tail->tmem_base), TMEM_COLS);
    ptx::tmem_relinquish();
  } else if (warp == 2) {
    // segment starts + exclusive scan of m-tiles per slot (warp-shuffle scan, 32 slots a step)
    int carry = 0;
    for (int base = 0; base < E_loc; base += 32) {
      const int e = base + lane;
      int lo = 0, hi = 0;
      if (e < E_loc) {
        lo = offsets[e];
        hi = offsets[e + 1];
        tail->off[e] = lo;
      }
      const int mt = (hi - lo + BM - 1) / BM;
      int inc = mt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
      }
      if (e < E_loc) tail->cum[e] = carry + inc - mt;
      carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) {
      tail->cum[E_loc] = carry;
      tail->off[E_loc] = offsets[E_loc];
      tail->total_m_tiles = carry;
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();

  const uint32_t tmem_base = tail->tmem_base;
  const int total_tiles = tail->total_m_tiles * NB;

  if (warp == 0) {
    // ================================================================ TMA producer
    if (lane == 0) {
      const uint64_t pol_a = ptx::policy_evict_last();    // activations are re-read by every n-block
      const uint64_t pol_b = ptx::policy_evict_first();   // each weight byte is needed once (per wave)
      TileCursor cur;
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        int m_blk, n_blk;
        cur.decode(tail, tile, NB, m_blk, n_blk);
        const int e = cur.e;
        const int row0 = tail->off[e] + m_blk * BM;
        const int n0 = n_blk * BN_OUT;
        for (int kb = 0; kb < KB; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->empty[stage]), phase ^ 1u);
          const uint32_t full = ptx::smem_u32(&tail->full[stage]);
          ptx::mbar_arrive_expect_tx(full, STAGE_BYTES);
          const uint32_t a_s = ptx::smem_u32(smem + (size_t)stage * STAGE_BYTES);
          const uint32_t b_s = a_s + A_BYTES;
          const int k0 = kb * BK;
          ptx::tma_load_2d(a_s, &tmA, full, k0, row0, pol_a);
          if (kGateUp) {
            ptx::tma_load_3d(b_s + 0 * B_ATOM_BYTES, &tmB0, full, n0, k0, e, pol_b);
            ptx::tma_load_3d(b_s + 1 * B_ATOM_BYTES, &tmB0, full, n0 + 64, k0, e, pol_b);
            ptx::tma_load_3d(b_s + 2 * B_ATOM_BYTES, &tmB1, full, n0, k0, e, pol_b);
            ptx::tma_load_3d(b_s + 3 * B_ATOM_BYTES, &tmB1, full, n0 + 64, k0, e, pol_b);
          } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
              ptx::tma_load_3d(b_s + j * B_ATOM_BYTES, &tmB0, full, n0 + 64 * j, k0, e, pol_b);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ UMMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16_f32(BM, UMMA_N, /*a_mn=*/false, /*b_mn=*/true);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&tail->tempty[acc]), acc_phase ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * UMMA_N;
        for (int kb = 0; kb < KB; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->full[stage]), phase);
          ptx::tc_fence_after();
          const uint32_t a_s = ptx::smem_u32(smem + (size_t)stage * STAGE_BYTES);
          const uint32_t b_s = a_s + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k) {
            // A: K-major SW128 -> advance 16 elements = 32 bytes inside the 128-byte row
            const uint64_t da = ptx::make_smem_desc_sw128(a_s + k * (UMMA_K * 2), 16, 1024);
            // B: MN-major SW128 -> 16 K-rows = 2 swizzle atoms of 1024 B; next 64 N-columns at LBO
            const uint64_t db = ptx::make_smem_desc_sw128(b_s + k * (UMMA_K * 128), B_ATOM_BYTES, 1024);
            ptx::umma_bf16(d_tmem, da, db, idesc, (uint32_t)((kb | k) != 0));
          }
          ptx::umma_commit(ptx::smem_u32(&tail->empty[stage]));   // frees the smem stage when MMAs retire
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        ptx::umma_commit(ptx::smem_u32(&tail->tfull[acc]));       // accumulator ready for the epilogue
      }
    }
  } else {
    // ================================================================ epilogue (warps 2..5)
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    TileCursor cur;
    int it = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
      int m_blk, n_blk;
      cur.decode(tail, tile, NB, m_blk, n_blk);
      const int e = cur.e;
      const int seg_end = tail->off[e + 1];
      const int grow = tail->off[e] + m_blk * BM + q * 32 + lane;
      const bool row_ok = grow < seg_end;
      const int n0 = n_blk * BN_OUT;
      const int acc = it & 1;
      const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
      ptx::mbar_wait(ptx::smem_u32(&tail->tfull[acc]), acc_phase);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)acc * UMMA_N;
      __nv_bfloat16* orow = out + (size_t)grow * ld_out + n0;
      if (kGateUp) {
#pragma unroll 1
        for (int c = 0; c < 4; ++c) {
          uint32_t g[32], u[32];
          ptx::tmem_ld_32x32(taddr + c * 32, g);
          ptx::tmem_ld_32x32(taddr + 128 + c * 32, u);
          ptx::tmem_ld_wait();
          uint32_t h[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const float g0 = __uint_as_float(g[2 * i]), g1 = __uint_as_float(g[2 * i + 1]);
            const float u0 = __uint_as_float(u[2 * i]), u1 = __uint_as_float(u[2 * i + 1]);
            const float h0 = __fdividef(g0, 1.0f + __expf(-g0)) * u0;
            const float h1 = __fdividef(g1, 1.0f + __expf(-g1)) * u1;
            h[i] = pack2_bf16(h0, h1);
          }
          if (row_ok && n0 + c * 32 < n_total) {
            uint4* dst = reinterpret_cast<uint4*>(orow + c * 32);
#pragma unroll
            for (int v = 0; v < 4; ++v) dst[v] = make_uint4(h[4 * v], h[4 * v + 1], h[4 * v + 2], h[4 * v + 3]);
          }
        }
      } else {
#pragma unroll 1
        for (int c = 0; c < 8; ++c) {
          uint32_t a[32];
          ptx::tmem_ld_32x32(taddr + c * 32, a);
          ptx::tmem_ld_wait();
          if (row_ok && n0 + c * 32 < n_total) {
            uint4* dst = reinterpret_cast<uint4*>(orow + c * 32);
#pragma unroll
            for (int v = 0; v < 4; ++v) {
              uint4 o;
              o.x = pack2_bf16(__uint_as_float(a[8 * v + 0]), __uint_as_float(a[8 * v + 1]));
              o.y = pack2_bf16(__uint_as_float(a[8 * v + 2]), __uint_as_float(a[8 * v + 3]));
              o.z = pack2_bf16(__uint_as_float(a[8 * v + 4]), __uint_as_float(a[8 * v + 5]));
              o.w = pack2_bf16(__uint_as_float(a[8 * v + 6]), __uint_as_float(a[8 * v + 7]));
              dst[v] = o;
            }
          }
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&tail->tempty[acc]));
    }
  }

  // ------------------------------------------------------------------ teardown
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, TMEM_COLS);
  }
}

// ---------------------------------------------------------------------------------------
// TMA tensor maps (host).  cuTensorMapEncodeTiled is a driver entry point fetched through
// the runtime, so libvibe.so does not link libcuda.  Maps are cached for the process
// lifetime, keyed by (pointer, shape): weights and workspaces are long-lived in serving.
// ---------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

struct MapKey {
  const void* ptr;
  uint64_t d0, d1, d2;
  uint32_t b0, b1;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b0 == o.b0 && b1 == o.b1;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = reinterpret_cast<size_t>(k.ptr);
    h = h * 1315423911u ^ k.d0;
    h = h * 1315423911u ^ k.d1;
    h = h * 1315423911u ^ k.d2;
    h = h * 1315423911u ^ ((uint64_t)k.b0 << 32 | k.b1);
    return h;
  }
};
std::mutex g_map_mu;
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// rank 2: dims (d0 inner, d1); rank 3: dims (d0 inner, d1, d2).  bf16, 128-byte swizzle.
vibe_status get_tensor_map(const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box0, uint32_t box1,
                           CUtensorMap* out) {
  MapKey key{ptr, d0, d1, d2, box0, box1};
  {
    std::lock_guard<std::mutex> lk(g_map_mu);
    auto it = g_maps.find(key);
    if (it != g_maps.end()) {
      *out = it->second;
      return VIBE_OK;
    }
  }
  EncodeTiledFn enc = get_encode_fn();
  VIBE_REQUIRE(enc != nullptr, VIBE_ERR_CUDA, "cuTensorMapEncodeTiled entry point unavailable (no CUDA driver?)");
  const bool r3 = d2 > 0;
  cuuint64_t dims[3] = {d0, d1, r3 ? d2 : 1};
  cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
  cuuint32_t box[3] = {box0, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, r3 ? 3 : 2, const_cast<void*>(ptr), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  VIBE_REQUIRE(r == CUDA_SUCCESS, VIBE_ERR_CUDA,
               "cuTensorMapEncodeTiled failed (CUresult %d) ptr=%p dims=(%llu,%llu,%llu) box=(%u,%u)", (int)r, ptr,
               (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, box0, box1);
  {
    std::lock_guard<std::mutex> lk(g_map_mu);
    if (g_maps.size() > 4096) g_maps.clear();
    g_maps[key] = m;
  }
  *out = m;
  return VIBE_OK;
}

}  // namespace

vibe_status grouped_ffn_impl(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                             const void* W1, const void* W3, const void* W2, void* H_ws, void* Y,
                             cudaStream_t st) {
  CUtensorMap tmX, tmH, tmW1, tmW3, tmW2;
  vibe_status s;
  if ((s = get_tensor_map(Xp, d, R_cap, 0, BK, BM, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(H_ws, f, R_cap, 0, BK, BM, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W1, f, d, E_loc, 64, BK, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W3, f, d, E_loc, 64, BK, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W2, d, f, E_loc, 64, BK, &tmW2)) != VIBE_OK) return s;
  static std::once_flag once;
  static cudaError_t attr_err = cudaSuccess;
  std::call_once(once, [] {
    attr_err = cudaFuncSetAttribute(ffn_gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)SMEM_BYTES);
    if (attr_err == cudaSuccess)
      attr_err = cudaFuncSetAttribute(ffn_gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)SMEM_BYTES);
  });
  VIBE_REQUIRE(attr_err == cudaSuccess, VIBE_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %zu) failed: %s",
               SMEM_BYTES, cudaGetErrorString(attr_err));
  const int grid = num_sms();
  ffn_gemm_kernel<true><<<grid, NUM_THREADS, SMEM_BYTES, st>>>(tmX, tmW1, tmW3, offsets, E_loc, f, d,
                                                               reinterpret_cast<__nv_bfloat16*>(H_ws), f);
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<gate_up>");
  ffn_gemm_kernel<false><<<grid, NUM_THREADS, SMEM_BYTES, st>>>(tmH, tmW2, tmW2, offsets, E_loc, d, f,
                                                                reinterpret_cast<__nv_bfloat16*>(Y), d);
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<down>");
  return VIBE_OK;
}

vibe_status grouped_ffn_check(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                              const void* W1, const void* W3, const void* W2, void* H_ws, void* Y) {
  VIBE_REQUIRE(E_loc >= 1 && R_cap >= 1 && d >= 1 && f >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_grouped_ffn: bad sizes E_loc=%d R_cap=%d d=%d f=%d", E_loc, R_cap, d, f);
  VIBE_REQUIRE(Xp && offsets && W1 && W3 && W2 && H_ws && Y, VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn: NULL tensor");
  VIBE_REQUIRE(d % 64 == 0 && f % 64 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_grouped_ffn: d and f must be multiples of 64 (d=%d f=%d)", d, f);
  VIBE_REQUIRE(E_loc <= MAX_SLOTS, VIBE_ERR_UNSUPPORTED, "vibe_grouped_ffn: E_loc > %d not implemented", MAX_SLOTS);
  VIBE_REQUIRE(aligned16(Xp) && aligned16(W1) && aligned16(W3) && aligned16(W2) && aligned16(H_ws) && aligned16(Y),
               VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn: all tensors must be 16-byte aligned");
  return VIBE_OK;
}

}  // namespace vibe

extern "C" vibe_status vibe_grouped_ffn(const void* Xp, const int32_t* offsets, int32_t E_loc, int32_t R_cap,
                                        int32_t d, int32_t f, const void* W1, const void* W3, const void* W2,
                                        void* H_ws, void* Y, void* ws, size_t ws_bytes, void* stream) {
  using namespace vibe;
  (void)ws;
  (void)ws_bytes;
  clear_error();
  vibe_status s = grouped_ffn_check(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Y);
  if (s != VIBE_OK) return s;
  return grouped_ffn_impl(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Y,
                          reinterpret_cast<cudaStream_t>(stream));
}
