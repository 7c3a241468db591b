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

// ---------------------------------------------------------------------------------------------------------
// Block-scaled variant (readings Q5-Q7): one UE8M0 scale 2^e per `block` (32 | 128) consecutive K elements of a
// row, e = the smallest integer with amax <= 448 * 2^e (448 = 1.75 * 2^8: e = x - 8, +1 when the mantissa of
// amax = m * 2^x exceeds 1.75), clamped to >= -127, 0 for an all-zero block; stored byte e + 127, one byte per
// 32 elements; code = e4m3_rn(x * 2^-e) (the scaling is exact).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int mx_exponent(float amax) {
  const uint32_t bits = __float_as_uint(amax);
  const int ex = (int)(bits >> 23) - 127 - 8 + ((bits & 0x7fffffu) > 0x600000u ? 1 : 0);
  return bits == 0u ? 0 : max(ex, -127);
}
__device__ __forceinline__ float mx_inv_scale(int ex) { return __uint_as_float((uint32_t)(127 - ex) << 23); }

// byte offset of the scale of (row r, 32-block b) in the token layout [K/128][32][Rb] words (vibe.h)
__device__ __forceinline__ size_t mx_token_sf_offset(int r, int b, int Rb) {
  return ((size_t)((b >> 2) * 32 + (r & 31)) * (size_t)Rb + (size_t)(r >> 5)) * 4 + (size_t)(b & 3);
}

// one warp per row; lane l holds the 16-byte vectors l, l + 32, ...: a 32-block is 4 neighbouring lanes of one
// vector round, a 128-block 16 of them
__global__ void __launch_bounds__(256) mx_quantize_rows_kernel(const __nv_bfloat16* __restrict__ X, int R, int d, int block,
                                                               uint8_t* __restrict__ Xq, uint8_t* __restrict__ sf,
                                                               int sf_tokens_layout, int Rb, const int32_t* __restrict__ ids,
                                                               const int32_t* __restrict__ emap, int k, int E, int E_loc) {
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
    uint2* dst = reinterpret_cast<uint2*>(Xq + (size_t)r * d);
    for (int v0 = lane; v0 - lane < vpr; v0 += 128) {          // warp-uniform trip count (shuffles inside)
      uint4 q[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) q[j] = (v0 + 32 * j < vpr) ? src[v0 + 32 * j] : make_uint4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t w[4] = {q[j].x, q[j].y, q[j].z, q[j].w};
        float amax = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i) amax = fmaxf(amax, fmaxf(fabsf(bf16_lo(w[i])), fabsf(bf16_hi(w[i]))));
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 1));
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 2));
        if (block == 128) {
          amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 4));
          amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 8));
        }
        const int ex = mx_exponent(amax);
        const float inv = mx_inv_scale(ex);
        uint32_t p[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) p[i] = ptx::pack2_e4m3(bf16_lo(w[i]) * inv, bf16_hi(w[i]) * inv);
        const int v = v0 + 32 * j;
        if (v < vpr) {
          dst[v] = make_uint2(p[0] | (p[1] << 16), p[2] | (p[3] << 16));
          if ((lane & 3) == 0) {
            const int b = v >> 2;
            sf[sf_tokens_layout ? mx_token_sf_offset(r, b, Rb) : (size_t)r * (d >> 5) + b] = (uint8_t)(ex + 127);
          }
        }
      }
    }
  }
}

// W [E,K,N] bf16 -> Wq [E,N,K] e4m3 + scales in the weight-chunk layouts (vibe.h).  One thread block per
// (32 features, `block` K elements, expert): the tile goes through shared memory transposed.
__global__ void __launch_bounds__(256) mx_pack_kernel(const __nv_bfloat16* __restrict__ W, int K, int N, int block, int role,
                                                      uint8_t* __restrict__ Wq, uint8_t* __restrict__ sf) {
  __shared__ float tile[128][33];
  const int e = blockIdx.z;
  const __nv_bfloat16* src = W + (size_t)e * K * N;
  uint8_t* dst = Wq + (size_t)e * K * N;
  const int n0 = blockIdx.x * 32, k0 = blockIdx.y * block;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
  for (int kk = ty; kk < block; kk += 8) tile[kk][tx] = __bfloat162float(src[(size_t)(k0 + kk) * N + n0 + tx]);
  __syncthreads();
  const int KS = K >> 7;
  for (int nn = ty; nn < 32; nn += 8) {
    const int n = n0 + nn;
    float v[4];
    float amax = 0.0f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      v[j] = (32 * j < block) ? tile[tx + 32 * j][nn] : 0.0f;
      amax = fmaxf(amax, fabsf(v[j]));
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const int ex = mx_exponent(amax);
    const float inv = mx_inv_scale(ex);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (32 * j >= block) break;
      dst[(size_t)n * K + k0 + tx + 32 * j] = (uint8_t)(ptx::pack2_e4m3(v[j] * inv, 0.0f) & 0xffu);
      if (tx == 0) {
        const int b = (k0 >> 5) + j;
        size_t off;
        if (role == VIBE_MX_ROLE_DOWN)
          off = ((size_t)(e * KS + (b >> 2)) * (size_t)(N >> 7) + (size_t)(n >> 7)) * 512 + (size_t)(n & 31) * 16 +
                (size_t)((n & 127) >> 5) * 4 + (size_t)(b & 3);
        else
          off = ((size_t)(e * KS + (b >> 2)) * (size_t)(N >> 6) + (size_t)(n >> 6)) * 512 + (size_t)(n & 31) * 16 +
                (size_t)(((n & 63) >> 5) + (role == VIBE_MX_ROLE_UP ? 2 : 0)) * 4 + (size_t)(b & 3);
        sf[off] = (uint8_t)(ex + 127);
      }
    }
  }
}

// token scales [T][d/32] (row-major, as the row quantiser wrote them before the permutation) -> the token layout
// for the PERMUTED rows; padding rows and rows past the last segment get the byte 127 (scale 1)
__global__ void __launch_bounds__(256) mx_gather_row_sf_kernel(const uint32_t* __restrict__ tok_sf, const int32_t* __restrict__ row_to_assign,
                                                               const int32_t* __restrict__ offsets, int E_loc, int k, int R_cap,
                                                               int KS, int Rb, uint32_t* __restrict__ out) {
  const int R = __ldg(offsets + E_loc);
  const long long total = (long long)R_cap * KS;
  for (long long idx = (long long)blockIdx.x * 256 + threadIdx.x; idx < total; idx += (long long)gridDim.x * 256) {
    const int s = (int)(idx / R_cap), r = (int)(idx - (long long)s * R_cap);
    uint32_t w = 0x7f7f7f7fu;
    if (r < R) {
      const int i = __ldg(row_to_assign + r);
      if (i >= 0) w = __ldg(tok_sf + (size_t)(i / k) * KS + s);
    }
    out[(size_t)(s * 32 + (r & 31)) * Rb + (r >> 5)] = w;
  }
}

}  // namespace

vibe_status mx_gather_row_sf(const void* tok_sf, const int32_t* row_to_assign, const int32_t* offsets, int E_loc, int k,
                             int R_cap, int d, void* out, cudaStream_t st) {
  const long long total = (long long)R_cap * (d / 128);
  int blocks = (int)((total + 255) / 256 < (long long)num_sms() * 16 ? (total + 255) / 256 : (long long)num_sms() * 16);
  if (blocks < 1) blocks = 1;
  mx_gather_row_sf_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const uint32_t*>(tok_sf), row_to_assign, offsets, E_loc, k,
                                                  R_cap, d / 128, mx_row_blocks(R_cap), reinterpret_cast<uint32_t*>(out));
  VIBE_LAUNCH_CHECK("mx_gather_row_sf_kernel");
  return VIBE_OK;
}

vibe_status mx_quantize_rows(const void* X, int R, int d, int block, void* Xq, void* sf, int sf_layout, int R_cap,
                             const int32_t* ids, const int32_t* emap, int k, int E, int E_loc, cudaStream_t st) {
  if (R == 0) return VIBE_OK;
  int blocks = (R + 7) / 8;
  if (blocks > num_sms() * 16) blocks = num_sms() * 16;
  mx_quantize_rows_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const __nv_bfloat16*>(X), R, d, block,
                                                  reinterpret_cast<uint8_t*>(Xq), reinterpret_cast<uint8_t*>(sf), sf_layout,
                                                  mx_row_blocks(R_cap), ids, emap, k, E, E_loc);
  VIBE_LAUNCH_CHECK("mx_quantize_rows_kernel");
  return VIBE_OK;
}

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

extern "C" size_t vibe_mxfp8_sf_bytes(int32_t which, int32_t rows, int32_t K, int32_t E_loc) {
  using namespace vibe;
  if (rows < 1 || K < 128 || K % 128 != 0 || E_loc < 1) return 0;
  switch (which) {
    case VIBE_MX_SF_ROWMAJOR: return (size_t)rows * (K / 32);
    case VIBE_MX_SF_TOKENS: return (size_t)(K / 128) * 32 * (size_t)mx_row_blocks(rows) * 4;
    case VIBE_MX_SF_GATE_UP: return rows % 64 ? 0 : (size_t)E_loc * (K / 128) * (rows / 64) * 512;
    case VIBE_MX_SF_DOWN: return rows % 128 ? 0 : (size_t)E_loc * (K / 128) * (rows / 128) * 512;
    default: return 0;
  }
}

extern "C" vibe_status vibe_mxfp8_quantize_rows(const void* X, int32_t R, int32_t d, int32_t block, void* Xq, void* sf,
                                                int32_t sf_layout, int32_t R_cap, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(R >= 0 && d >= 128 && d % 128 == 0, VIBE_ERR_INVALID_ARG, "vibe_mxfp8_quantize_rows: bad sizes R=%d d=%d (d % 128 == 0)", R, d);
  VIBE_REQUIRE(block == 32 || block == 128, VIBE_ERR_INVALID_ARG, "vibe_mxfp8_quantize_rows: block must be 32 or 128 (got %d)", block);
  VIBE_REQUIRE(sf_layout == VIBE_MX_SF_ROWMAJOR || (sf_layout == VIBE_MX_SF_TOKENS && R_cap >= R), VIBE_ERR_INVALID_ARG,
               "vibe_mxfp8_quantize_rows: sf_layout must be ROWMAJOR, or TOKENS with R_cap >= R");
  if (R == 0) return VIBE_OK;
  VIBE_REQUIRE(X && Xq && sf, VIBE_ERR_INVALID_ARG, "vibe_mxfp8_quantize_rows: NULL tensor");
  VIBE_REQUIRE(aligned16(X) && aligned16(Xq), VIBE_ERR_INVALID_ARG, "vibe_mxfp8_quantize_rows: X / Xq must be 16-byte aligned");
  return mx_quantize_rows(X, R, d, block, Xq, sf, sf_layout, sf_layout == VIBE_MX_SF_TOKENS ? R_cap : R, nullptr, nullptr, 0, 0,
                          0, reinterpret_cast<cudaStream_t>(stream));
}

extern "C" vibe_status vibe_mxfp8_pack_weights(const void* W, int32_t E_loc, int32_t K, int32_t N, int32_t block,
                                               int32_t role, void* Wq, void* sf, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(E_loc >= 1 && K >= 128 && N >= 128 && K % 128 == 0 && N % 128 == 0, VIBE_ERR_INVALID_ARG,
               "vibe_mxfp8_pack_weights: bad sizes E_loc=%d K=%d N=%d (K, N multiples of 128)", E_loc, K, N);
  VIBE_REQUIRE(block == 32 || block == 128, VIBE_ERR_INVALID_ARG, "vibe_mxfp8_pack_weights: block must be 32 or 128 (got %d)", block);
  VIBE_REQUIRE(role == VIBE_MX_ROLE_DOWN || role == VIBE_MX_ROLE_GATE || role == VIBE_MX_ROLE_UP, VIBE_ERR_INVALID_ARG,
               "vibe_mxfp8_pack_weights: bad role %d", role);
  VIBE_REQUIRE(W && Wq && sf, VIBE_ERR_INVALID_ARG, "vibe_mxfp8_pack_weights: NULL tensor");
  VIBE_REQUIRE(E_loc <= 65535 && K / block <= 65535, VIBE_ERR_UNSUPPORTED, "vibe_mxfp8_pack_weights: shape too large");
  mx_pack_kernel<<<dim3(N / 32, K / block, E_loc), 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(
      reinterpret_cast<const __nv_bfloat16*>(W), K, N, block, role, reinterpret_cast<uint8_t*>(Wq), reinterpret_cast<uint8_t*>(sf));
  VIBE_LAUNCH_CHECK("mx_pack_kernel");
  return VIBE_OK;
}
