// combine.cu -- a5: gate-weighted un-permute / combine (vibe_combine).
//   out[t,:] = bf16( sum_j topk_w[t,j] * Y[assign_to_row[t*k+j],:] ),  fp32, slot order.
// Token-major, one thread per 16-byte output vector(s), up to 4*VPT row loads in flight per
// thread.  HBM-bound: reads 2*R*d, writes 2*T*d bytes.  include/vibe.h, C1.
#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

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

// One thread per VPT 16-byte output vectors of one token (vectors v and v + vpr/2 of the
// same row when VPT == 2, so the k (row, weight) pairs are fetched once per thread; they are
// warp-uniform addresses -> one broadcast transaction, L1-resident after the first warp, and
// 16-byte vector loads when k % 4 == 0).  Non-resident slots are skipped with a warp-uniform
// branch (a warp never straddles tokens when vpr/VPT % 32 == 0; otherwise it merely diverges).
// No grid-stride loop and no block barrier: the grid covers T * vpr / VPT threads and the
// hardware scheduler keeps ~2048 threads x up to 4*VPT independent 16-byte loads in flight per SM.
// SCAT: Y holds gate-weighted rows in ASSIGNMENT order (vibe_grouped_ffn_scatter): slot j of
// token t reads row t*k + j with weight 1 when assign_to_row[t*k + j] >= 0 (topk_w unused).
template <int VPT, bool K4, bool SCAT>
__global__ void __launch_bounds__(256) combine_kernel(const __nv_bfloat16* __restrict__ Y,
                                                      const int32_t* __restrict__ assign_to_row,
                                                      const float* __restrict__ topk_w, int T, int k, int d,
                                                      __nv_bfloat16* __restrict__ out) {
  const int vpr = d >> 3;            // 16-byte vectors per row
  const int per_row = vpr / VPT;     // threads per row
  ptx::griddep_wait();               // launched as a programmatic dependent of the kernel that writes Y
  const long long g = (long long)blockIdx.x * 256 + threadIdx.x;
  if (g >= (long long)T * per_row) return;
  const int t = (int)(g / per_row);
  const int v0 = (int)(g - (long long)t * per_row);
  const int32_t* a2r = assign_to_row + (size_t)t * k;
  const float* wt = topk_w + (size_t)t * k;
  float acc[VPT][8];
#pragma unroll
  for (int q = 0; q < VPT; ++q)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[q][i] = 0.0f;
  for (int j0 = 0; j0 < k; j0 += 4) {
    int r[4];
    float w[4];
    if (K4) {
      const int4 rr = __ldg(reinterpret_cast<const int4*>(a2r + j0));
      r[0] = rr.x; r[1] = rr.y; r[2] = rr.z; r[3] = rr.w;
      if (!SCAT) {
        const float4 ww = __ldg(reinterpret_cast<const float4*>(wt + j0));
        w[0] = ww.x; w[1] = ww.y; w[2] = ww.z; w[3] = ww.w;
      }
    } else {
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        r[jj] = (j0 + jj < k) ? __ldg(a2r + j0 + jj) : -1;
        if (!SCAT) w[jj] = (j0 + jj < k) ? __ldg(wt + j0 + jj) : 0.0f;
      }
    }
    if (SCAT) {
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        r[jj] = (r[jj] >= 0) ? t * k + j0 + jj : -1;
        w[jj] = 1.0f;
      }
    }
    if ((r[0] & r[1] & r[2] & r[3]) < 0) continue;   // all four slots non-resident (sign bits)
    uint4 val[4][VPT];
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
#pragma unroll
      for (int q = 0; q < VPT; ++q) val[jj][q] = make_uint4(0, 0, 0, 0);
      if (r[jj] >= 0) {
        const uint4* src = reinterpret_cast<const uint4*>(Y + (size_t)r[jj] * d) + v0;
#pragma unroll
        for (int q = 0; q < VPT; ++q) val[jj][q] = ld_nc_v4(src + q * per_row);
      }
    }
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
      if (r[jj] >= 0) {   // slot order j = 0..k-1, skipped slots contribute nothing
#pragma unroll
        for (int q = 0; q < VPT; ++q) fma_bf16x8(acc[q], val[jj][q], w[jj]);
      }
    }
  }
#pragma unroll
  for (int q = 0; q < VPT; ++q) {
    uint4 o;
    o.x = pack_bf16x2(acc[q][0], acc[q][1]);
    o.y = pack_bf16x2(acc[q][2], acc[q][3]);
    o.z = pack_bf16x2(acc[q][4], acc[q][5]);
    o.w = pack_bf16x2(acc[q][6], acc[q][7]);
    st_na_v4(reinterpret_cast<uint4*>(out + (size_t)t * d) + v0 + q * per_row, o);
  }
}

}  // namespace
}  // namespace vibe

namespace vibe {
namespace {
vibe_status combine_impl(const char* who, const void* Y, const int32_t* assign_to_row, const float* topk_w, int T,
                         int k, int d, void* out, void* stream, bool scat) {
  clear_error();
  VIBE_REQUIRE(T >= 0 && k >= 1 && d >= 8, VIBE_ERR_INVALID_ARG, "%s: bad sizes T=%d k=%d d=%d", who, T, k, d);
  VIBE_REQUIRE(d % 8 == 0, VIBE_ERR_INVALID_ARG, "%s: d %% 8 != 0", who);
  VIBE_REQUIRE(k <= 32, VIBE_ERR_UNSUPPORTED, "%s: k > 32 not implemented (vibe_route_topk limit)", who);
  if (T == 0) return VIBE_OK;
  VIBE_REQUIRE(Y && assign_to_row && (scat || topk_w) && out, VIBE_ERR_INVALID_ARG, "%s: NULL tensor", who);
  VIBE_REQUIRE(aligned16(Y) && aligned16(out), VIBE_ERR_INVALID_ARG, "%s: Y / out must be 16-byte aligned", who);
  VIBE_REQUIRE((int64_t)T * k < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "%s: T*k >= 2^31", who);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int vpr = d / 8;
  const __nv_bfloat16* Yb = reinterpret_cast<const __nv_bfloat16*>(Y);
  __nv_bfloat16* ob = reinterpret_cast<__nv_bfloat16*>(out);
  const int vpt = (vpr % 2 == 0) ? 2 : 1;
  const bool k4 = (k % 4 == 0) && aligned16(assign_to_row) && (scat || aligned16(topk_w));
  const long long threads = (long long)T * (vpr / vpt);
  const long long blocks = (threads + 255) / 256;
  VIBE_REQUIRE(blocks < (1ll << 31), VIBE_ERR_UNSUPPORTED, "%s: T*d too large for one launch", who);
  const unsigned gb = (unsigned)blocks;
  cudaError_t launch_err = cudaSuccess;
#define VIBE_COMBINE_CASE(V, K, S)                                                              \
  if (vpt == V && k4 == K && scat == S)                                                         \
    launch_err = launch_pdl(combine_kernel<V, K, S>, dim3(gb), dim3(256), 0, st, Yb, assign_to_row, topk_w, T, k, d, ob);
  VIBE_COMBINE_CASE(2, true, false)
  VIBE_COMBINE_CASE(2, false, false)
  VIBE_COMBINE_CASE(1, true, false)
  VIBE_COMBINE_CASE(1, false, false)
  VIBE_COMBINE_CASE(2, true, true)
  VIBE_COMBINE_CASE(2, false, true)
  VIBE_COMBINE_CASE(1, true, true)
  VIBE_COMBINE_CASE(1, false, true)
#undef VIBE_COMBINE_CASE
  VIBE_REQUIRE(launch_err == cudaSuccess, VIBE_ERR_CUDA, "combine_kernel launch failed: %s", cudaGetErrorString(launch_err));
  VIBE_LAUNCH_CHECK("combine_kernel");
  return VIBE_OK;
}
}  // namespace
}  // namespace vibe

extern "C" vibe_status vibe_combine(const void* Y, const int32_t* assign_to_row, const float* topk_w, int32_t T,
                                    int32_t k, int32_t d, void* out, void* stream) {
  return vibe::combine_impl("vibe_combine", Y, assign_to_row, topk_w, T, k, d, out, stream, false);
}

extern "C" vibe_status vibe_combine_scattered(const void* Yw, const int32_t* assign_to_row, int32_t T, int32_t k,
                                              int32_t d, void* out, void* stream) {
  return vibe::combine_impl("vibe_combine_scattered", Yw, assign_to_row, nullptr, T, k, d, out, stream, true);
}
