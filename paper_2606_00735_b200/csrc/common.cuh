// common.cuh -- shared plumbing of libvibe.so (host error state, launch accounting, small
// device helpers).  CUDA path only: nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>
#include <stdarg.h>

#include "../../include/vibe.h"

namespace vibe {

// ---- host-side error state (thread-local) -------------------------------------------
void set_error(const char* fmt, ...);
void clear_error();
void count_launch(int n = 1);
int num_sms();            // of the current device
constexpr int kMaxDevices = 64;
constexpr size_t kProfileFlushBytes = (size_t)256 << 20;   // L2 flush region at the END of a VIBE_WS_PROFILE workspace (2 x the 126 MB L2)
int current_device();     // ordinal in [0, kMaxDevices)

#define VIBE_REQUIRE(cond, status, ...)         \
  do {                                          \
    if (!(cond)) {                              \
      ::vibe::set_error(__VA_ARGS__);           \
      return (status);                          \
    }                                           \
  } while (0)

#define VIBE_CUDA(call)                                                                   \
  do {                                                                                    \
    cudaError_t e__ = (call);                                                             \
    if (e__ != cudaSuccess) {                                                             \
      ::vibe::set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, \
                        __LINE__);                                                        \
      return VIBE_ERR_CUDA;                                                               \
    }                                                                                     \
  } while (0)

// after a <<<>>> launch
#define VIBE_LAUNCH_CHECK(name)                                                             \
  do {                                                                                      \
    cudaError_t e__ = cudaGetLastError();                                                   \
    if (e__ != cudaSuccess) {                                                               \
      ::vibe::set_error("launch of %s failed: %s", name, cudaGetErrorString(e__));          \
      return VIBE_ERR_CUDA;                                                                 \
    }                                                                                       \
    ::vibe::count_launch();                                                                 \
  } while (0)

// ---- internal cross-file declarations -------------------------------------------------
struct LayerArena {
  size_t ids, w, offsets, r2a, a2r, Xp, H, Y, perm_ws, ffn_ws, total;
  int64_t R_cap;
};
LayerArena layer_arena(int T, int k, int E_loc, int d, int f);
size_t permute_ws_bytes(int T, int k, int E_loc);
vibe_status grouped_ffn_impl(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                             const void* W1, const void* W3, const void* W2, void* H_ws, void* Y, cudaStream_t st,
                             const int32_t* row_to_assign = nullptr, const float* topk_w = nullptr, void* ws = nullptr,
                             size_t ws_bytes = 0, bool ws_zeroed = false);
size_t grouped_ffn_ws_bytes();   // split-K partial buffer + counters (VIBE_WS_FFN)
vibe_status grouped_ffn_zero_counters(void* ws, cudaStream_t st);   // what ws_zeroed = true promises
vibe_status grouped_ffn_fp8_impl(const void* Xq, const float* row_scale, const int32_t* offsets, int E_loc, int R_cap,
                                 int d, int f, const void* W1q, const float* s1, const void* W3q, const float* s3,
                                 const void* W2q, const float* s2, const float* h_scale, void* Hq, void* Y,
                                 cudaStream_t st, void* ws = nullptr, size_t ws_bytes = 0, bool ws_zeroed = false);
vibe_status grouped_ffn_mxfp8_impl(const void* Xq, const void* xsf, const int32_t* offsets, int E_loc, int R_cap, int d,
                                   int f, const void* W1q, const void* W3q, const void* sf13, const void* W2q,
                                   const void* sf2, void* Hq, void* hsf, void* Y, cudaStream_t st, void* ws = nullptr,
                                   size_t ws_bytes = 0, bool ws_zeroed = false);
// words per (K stage, lane) row of a token-scale array [K/128][32][Rb]: the 32-row blocks of R_cap rows, rounded up to
// a 16-byte row pitch (a TMA global stride; the kernel only fetches boxes of 4 row blocks that start on a multiple of 4,
// so a box is entirely inside or entirely outside the tensor)
static inline int mx_row_blocks(int R_cap) { return (((R_cap + 31) / 32) + 3) & ~3; }
vibe_status grouped_ffn_limits(const char* who, int E_loc, int d, int f, const void* W1, const void* W3, const void* W2);
vibe_status grouped_ffn_check(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                              const void* W1, const void* W3, const void* W2, void* H_ws, void* Y);

vibe_status fp8_gather_row_scales(const float* tok_scale, const int32_t* row_to_assign, const int32_t* offsets, int E_loc,
                                  int k, int R_cap, float* row_scale, cudaStream_t st);
vibe_status fp8_quantize_resident_tokens(const void* X, int T, int d, void* Xq, float* tok_scale, const int32_t* ids,
                                         const int32_t* emap, int k, int E, int E_loc, cudaStream_t st);
vibe_status mx_gather_row_sf(const void* tok_sf, const int32_t* row_to_assign, const int32_t* offsets, int E_loc, int k,
                             int R_cap, int d, void* out, cudaStream_t st);
vibe_status mx_quantize_rows(const void* X, int R, int d, int block, void* Xq, void* sf, int sf_layout, int R_cap,
                             const int32_t* ids, const int32_t* emap, int k, int E, int E_loc, cudaStream_t st);
// Launch with the programmatic-stream-serialization attribute (the kernel calls ptx::griddep_wait before it reads
// what the preceding kernel of the stream wrote).
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = grid;
  lc.blockDim = block;
  lc.dynamicSmemBytes = smem;
  lc.stream = st;
  lc.attrs = attr;
  lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kernel, KArgs(args)...);
}

struct LayerArenaFp8 {
  size_t ids, w, offsets, r2a, a2r, Xq, tok_scale, Xpq, row_scale, Hq, Y, perm_ws, ffn_ws, total;
  int64_t R_cap;
};
LayerArenaFp8 layer_arena_fp8(int T, int k, int E_loc, int d, int f);
struct LayerArenaMx {
  size_t ids, w, offsets, r2a, a2r, Xq, tok_sf, Xpq, xsf, Hq, hsf, Y, perm_ws, ffn_ws, total;
  int64_t R_cap;
};
LayerArenaMx layer_arena_mx(int T, int k, int E_loc, int d, int f);
constexpr int kMxRowAlign = 64;   // vibe_permute align of the block-scaled path: token tiles start on an even scale row block

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- device helpers ---------------------------------------------------------------------
__device__ __forceinline__ uint4 ld_nc_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void st_na_v4(void* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
}

}  // namespace vibe
