// combine.cu -- a5: gate-weighted un-permute / combine (vibe_combine).
//   out[t,:] = bf16( sum_j topk_w[t,j] * Y[assign_to_row[t*k+j],:] ),  fp32, slot order.
// Token-major: one CTA iteration per token, 16-byte vectors, up to k row loads in flight
// per thread.  HBM-bound: reads 2*R*d, writes 2*T*d bytes.  include/vibe.h, C1.
#include "common.cuh"

namespace vibe {
namespace {

constexpr int kMaxK = 32;

__device__ __forceinline__ void fma_bf16x8(float (&acc)[8], const uint4& v, float w) {
  const uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    acc[2 * i + 0] = fmaf(w, __uint_as_float(u[i] << 16), acc[2 * i + 0]);
    acc[2 * i + 1] = fmaf(w, __uint_as_float(u[i] & 0xffff0000u), acc[2 * i + 1]);
  }
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

template <int VEC>
__global__ void __launch_bounds__(256) combine_kernel(const __nv_bfloat16* __restrict__ Y,
                                                      const int32_t* __restrict__ assign_to_row,
                                                      const float* __restrict__ topk_w, int T, int k, int d,
                                                      __nv_bfloat16* __restrict__ out) {
  __shared__ int s_row[kMaxK];
  __shared__ float s_w[kMaxK];
  const int vec_per_row = d / 8;
  for (int t = blockIdx.x; t < T; t += gridDim.x) {
    __syncthreads();
    if (threadIdx.x < k) {
      s_row[threadIdx.x] = assign_to_row[(size_t)t * k + threadIdx.x];
      s_w[threadIdx.x] = topk_w[(size_t)t * k + threadIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < VEC; ++q) {
      const int v = threadIdx.x + q * 256;
      if (v >= vec_per_row) break;
      float acc[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) acc[i] = 0.0f;
      for (int j0 = 0; j0 < k; j0 += 4) {
        uint4 val[4];
        float w[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int j = j0 + jj;
          const int r = (j < k) ? s_row[j] : -1;
          w[jj] = (r >= 0) ? s_w[j] : 0.0f;
          val[jj] = (r >= 0) ? ld_nc_v4(reinterpret_cast<const uint4*>(Y + (size_t)r * d) + v)
                             : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) fma_bf16x8(acc, val[jj], w[jj]);
      }
      uint4 o;
      o.x = pack_bf16x2(acc[0], acc[1]);
      o.y = pack_bf16x2(acc[2], acc[3]);
      o.z = pack_bf16x2(acc[4], acc[5]);
      o.w = pack_bf16x2(acc[6], acc[7]);
      st_na_v4(reinterpret_cast<uint4*>(out + (size_t)t * d) + v, o);
    }
  }
}

}  // namespace
}  // namespace vibe

extern "C" vibe_status vibe_combine(const void* Y, const int32_t* assign_to_row, const float* topk_w, int32_t T,
                                    int32_t k, int32_t d, void* out, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(T >= 0 && k >= 1 && d >= 8, VIBE_ERR_INVALID_ARG, "vibe_combine: bad sizes T=%d k=%d d=%d", T, k, d);
  VIBE_REQUIRE(d % 8 == 0, VIBE_ERR_INVALID_ARG, "vibe_combine: d %% 8 != 0");
  VIBE_REQUIRE(k <= kMaxK, VIBE_ERR_UNSUPPORTED, "vibe_combine: k > %d not implemented", kMaxK);
  VIBE_REQUIRE(d <= 16384, VIBE_ERR_UNSUPPORTED, "vibe_combine: d > 16384 not implemented");
  if (T == 0) return VIBE_OK;
  VIBE_REQUIRE(Y && assign_to_row && topk_w && out, VIBE_ERR_INVALID_ARG, "vibe_combine: NULL tensor");
  VIBE_REQUIRE(aligned16(Y) && aligned16(out), VIBE_ERR_INVALID_ARG, "vibe_combine: Y / out must be 16-byte aligned");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int vec = (d / 8 + 255) / 256;
  const int blocks = T < num_sms() * 8 ? T : num_sms() * 8;
  const __nv_bfloat16* Yb = reinterpret_cast<const __nv_bfloat16*>(Y);
  __nv_bfloat16* ob = reinterpret_cast<__nv_bfloat16*>(out);
  if (vec <= 1)
    combine_kernel<1><<<blocks, 256, 0, st>>>(Yb, assign_to_row, topk_w, T, k, d, ob);
  else if (vec <= 2)
    combine_kernel<2><<<blocks, 256, 0, st>>>(Yb, assign_to_row, topk_w, T, k, d, ob);
  else if (vec <= 4)
    combine_kernel<4><<<blocks, 256, 0, st>>>(Yb, assign_to_row, topk_w, T, k, d, ob);
  else
    combine_kernel<8><<<blocks, 256, 0, st>>>(Yb, assign_to_row, topk_w, T, k, d, ob);
  VIBE_LAUNCH_CHECK("combine_kernel");
  return VIBE_OK;
}
