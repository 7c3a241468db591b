// fp8_quant.cu -- S8(f) f2: e4m3 quantisers feeding vibe_grouped_ffn_fp8 (readings Q1-Q3).
//   vibe_fp8_quantize_rows : bf16 [R,d]   -> e4m3 [R,d] + one scale per row (rowabsmax / 448)
//   vibe_fp8_pack_weights  : bf16 [E,K,N] -> e4m3 [E,N,K] (K contiguous: the re-layout is part of the one-time
//                            quantisation) + one scale per expert (absmax / 448)
// scale = binary32(amax / 448) (1 for an all-zero row / expert); code = e4m3_rn_satfinite(binary32(x / scale)).
#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }
__device__ __forceinline__ float scale_of(float amax) { return amax > 0.0f ? __fdiv_rn(amax, 448.0f) : 1.0f; }

// one warp per row, 16-byte vectors, 4 independent loads in flight per lane; the row is read twice (the second
// read is an L1/L2 hit)
// ids != NULL (expert-parallel shard): row t is skipped unless one of its k experts is resident -- the permutation
// never reads the rows of the other tokens.
__global__ void __launch_bounds__(256) fp8_quantize_rows_kernel(const __nv_bfloat16* __restrict__ X, int R, int d,
                                                                uint8_t* __restrict__ Xq, float* __restrict__ row_scale,
                                                                const int32_t* __restrict__ ids,
                                                                const int32_t* __restrict__ emap, int k, int E,
                                                                int E_loc) {
  const int lane = threadIdx.x & 31;
  const int vpr = d >> 3;
  for (int r = blockIdx.x * 8 + (threadIdx.x >> 5); r < R; r += gridDim.x * 8) {
    if (ids != nullptr) {
      bool res = false;
      for (int j = lane; j < k; j += 32) {
        const int e = __ldg(ids + (size_t)r * k + j);
        if (e >= 0 && e < E) {
          const int sl = emap ? __ldg(emap + e) : e;
          res |= (sl >= 0 && sl < E_loc);
        }
      }
      if (!__any_sync(0xffffffffu, res)) continue;
    }
    const uint4* src = reinterpret_cast<const uint4*>(X + (size_t)r * d);
    float amax = 0.0f;
    for (int v0 = lane; v0 < vpr; v0 += 128) {
      uint4 q[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) q[j] = (v0 + 32 * j < vpr) ? src[v0 + 32 * j] : make_uint4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t w[4] = {q[j].x, q[j].y, q[j].z, q[j].w};
#pragma unroll
        for (int i = 0; i < 4; ++i) amax = fmaxf(amax, fmaxf(fabsf(bf16_lo(w[i])), fabsf(bf16_hi(w[i]))));
      }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const float s = scale_of(amax);
    if (lane == 0) row_scale[r] = s;
    uint2* dst = reinterpret_cast<uint2*>(Xq + (size_t)r * d);
    for (int v0 = lane; v0 < vpr; v0 += 128) {
      uint4 q[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) q[j] = (v0 + 32 * j < vpr) ? src[v0 + 32 * j] : make_uint4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t w[4] = {q[j].x, q[j].y, q[j].z, q[j].w};
        uint32_t p[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) p[i] = ptx::pack2_e4m3(__fdiv_rn(bf16_lo(w[i]), s), __fdiv_rn(bf16_hi(w[i]), s));
        if (v0 + 32 * j < vpr) dst[v0 + 32 * j] = make_uint2(p[0] | (p[1] << 16), p[2] | (p[3] << 16));
      }
    }
  }
}

// absmax per expert: non-negative floats order like their bit patterns
__global__ void __launch_bounds__(256) fp8_absmax_kernel(const __nv_bfloat16* __restrict__ W, size_t per_expert,
                                                         unsigned int* __restrict__ amax_bits) {
  const int e = blockIdx.y;
  const uint4* src = reinterpret_cast<const uint4*>(W + (size_t)e * per_expert);
  const size_t nv = per_expert >> 3;
  float amax = 0.0f;
  for (size_t v = (size_t)blockIdx.x * 256 + threadIdx.x; v < nv; v += (size_t)gridDim.x * 256) {
    const uint4 q = src[v];
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) amax = fmaxf(amax, fmaxf(fabsf(bf16_lo(w[i])), fabsf(bf16_hi(w[i]))));
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  if ((threadIdx.x & 31) == 0) atomicMax(amax_bits + e, __float_as_uint(amax));
}

// [K,N] -> [N,K] through a 32 x 33 shared-memory tile, quantising on the way
__global__ void __launch_bounds__(256) fp8_pack_kernel(const __nv_bfloat16* __restrict__ W, int K, int N,
                                                       const float* __restrict__ amax, uint8_t* __restrict__ Wq) {
  __shared__ float tile[32][33];
  const int e = blockIdx.z;
  const float s = scale_of(amax[e]);
  const __nv_bfloat16* src = W + (size_t)e * K * N;
  uint8_t* dst = Wq + (size_t)e * K * N;
  const int n0 = blockIdx.x * 32, k0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
#pragma unroll
  for (int j = 0; j < 32; j += 8) {
    const int k = k0 + ty + j, n = n0 + tx;
    tile[ty + j][tx] = (k < K && n < N) ? __bfloat162float(src[(size_t)k * N + n]) : 0.0f;
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < 32; j += 8) {
    const int n = n0 + ty + j, k = k0 + tx;
    if (n < N && k < K) dst[(size_t)n * K + k] = (uint8_t)(ptx::pack2_e4m3(__fdiv_rn(tile[tx][ty + j], s), 0.0f) & 0xffu);
  }
}

__global__ void fp8_finish_scales_kernel(float* __restrict__ scale, int E) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < E) scale[e] = scale_of(scale[e]);
}

// row_scale[r] = scale of the token behind permuted row r (1 for padding rows and rows past the last segment)
__global__ void __launch_bounds__(256) fp8_gather_row_scales_kernel(const float* __restrict__ tok_scale,
                                                                    const int32_t* __restrict__ row_to_assign,
                                                                    const int32_t* __restrict__ offsets, int E_loc, int k,
                                                                    int R_cap, float* __restrict__ row_scale) {
  const int R = __ldg(offsets + E_loc);
  for (int r = blockIdx.x * 256 + threadIdx.x; r < R_cap; r += gridDim.x * 256) {
    float s = 1.0f;
    if (r < R) {
      const int i = __ldg(row_to_assign + r);
      if (i >= 0) s = __ldg(tok_scale + i / k);
    }
    row_scale[r] = s;
  }
}

}  // namespace

vibe_status fp8_gather_row_scales(const float* tok_scale, const int32_t* row_to_assign, const int32_t* offsets, int E_loc,
                                  int k, int R_cap, float* row_scale, cudaStream_t st) {
  int blocks = (R_cap + 255) / 256;
  if (blocks > num_sms() * 16) blocks = num_sms() * 16;
  if (blocks < 1) blocks = 1;
  fp8_gather_row_scales_kernel<<<blocks, 256, 0, st>>>(tok_scale, row_to_assign, offsets, E_loc, k, R_cap, row_scale);
  VIBE_LAUNCH_CHECK("fp8_gather_row_scales_kernel");
  return VIBE_OK;
}

vibe_status fp8_quantize_resident_tokens(const void* X, int T, int d, void* Xq, float* tok_scale, const int32_t* ids,
                                         const int32_t* emap, int k, int E, int E_loc, cudaStream_t st) {
  if (T == 0) return VIBE_OK;
  int blocks = (T + 7) / 8;
  if (blocks > num_sms() * 16) blocks = num_sms() * 16;
  fp8_quantize_rows_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const __nv_bfloat16*>(X), T, d,
                                                   reinterpret_cast<uint8_t*>(Xq), tok_scale, ids, emap, k, E, E_loc);
  VIBE_LAUNCH_CHECK("fp8_quantize_rows_kernel");
  return VIBE_OK;
}

}  // namespace vibe

extern "C" vibe_status vibe_fp8_quantize_rows(const void* X, int32_t R, int32_t d, void* Xq, float* row_scale,
                                              void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(R >= 0 && d >= 8 && d % 8 == 0, VIBE_ERR_INVALID_ARG, "vibe_fp8_quantize_rows: bad sizes R=%d d=%d", R, d);
  if (R == 0) return VIBE_OK;
  VIBE_REQUIRE(X && Xq && row_scale, VIBE_ERR_INVALID_ARG, "vibe_fp8_quantize_rows: NULL tensor");
  VIBE_REQUIRE(aligned16(X) && aligned16(Xq), VIBE_ERR_INVALID_ARG, "vibe_fp8_quantize_rows: X / Xq must be 16-byte aligned");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int blocks = (R + 7) / 8;
  if (blocks > num_sms() * 16) blocks = num_sms() * 16;
  fp8_quantize_rows_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const __nv_bfloat16*>(X), R, d,
                                                   reinterpret_cast<uint8_t*>(Xq), row_scale, nullptr, nullptr, 0, 0, 0);
  VIBE_LAUNCH_CHECK("fp8_quantize_rows_kernel");
  return VIBE_OK;
}

extern "C" vibe_status vibe_fp8_pack_weights(const void* W, int32_t E_loc, int32_t K, int32_t N, void* Wq, float* scale,
                                             void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(E_loc >= 1 && K >= 1 && N >= 1 && ((int64_t)K * N) % 8 == 0, VIBE_ERR_INVALID_ARG,
               "vibe_fp8_pack_weights: bad sizes E_loc=%d K=%d N=%d", E_loc, K, N);
  VIBE_REQUIRE(W && Wq && scale, VIBE_ERR_INVALID_ARG, "vibe_fp8_pack_weights: NULL tensor");
  VIBE_REQUIRE(aligned16(W), VIBE_ERR_INVALID_ARG, "vibe_fp8_pack_weights: W must be 16-byte aligned");
  VIBE_REQUIRE(E_loc <= 65535 && (K + 31) / 32 <= 65535, VIBE_ERR_UNSUPPORTED, "vibe_fp8_pack_weights: shape too large");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  VIBE_CUDA(cudaMemsetAsync(scale, 0, (size_t)E_loc * sizeof(float), st));
  const __nv_bfloat16* Wb = reinterpret_cast<const __nv_bfloat16*>(W);
  fp8_absmax_kernel<<<dim3(num_sms() * 2, E_loc), 256, 0, st>>>(Wb, (size_t)K * N, reinterpret_cast<unsigned int*>(scale));
  VIBE_LAUNCH_CHECK("fp8_absmax_kernel");
  fp8_pack_kernel<<<dim3((N + 31) / 32, (K + 31) / 32, E_loc), 256, 0, st>>>(Wb, K, N, scale,
                                                                              reinterpret_cast<uint8_t*>(Wq));
  VIBE_LAUNCH_CHECK("fp8_pack_kernel");
  fp8_finish_scales_kernel<<<(E_loc + 255) / 256, 256, 0, st>>>(scale, E_loc);
  VIBE_LAUNCH_CHECK("fp8_finish_scales_kernel");
  return VIBE_OK;
}
