// profile.cu -- a6: per-expert latency profile f(n) of the grouped FFN (vibe_profile_expert_latency).
// "Each GPU is warmed to steady-state operating conditions and profiled independently using
// the fused MoE kernel across a range of token counts.  This produces a function f_g(n)"
// (Algorithm 1 Phase 1, L439-L443; protocol L335).  DESIGN.md M1-M4.
#include <algorithm>
#include <vector>

#include "common.cuh"

namespace vibe {
namespace {
// arbitrary finite activations in (-1,1): latency does not depend on the values
__global__ void fill_pattern_kernel(__nv_bfloat16* p, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    uint32_t h = (uint32_t)i * 2654435761u;
    h ^= h >> 15;
    h *= 2246822519u;
    h ^= h >> 13;
    p[i] = __float2bfloat16_rn(((int)(h & 0xffff) - 32768) * (1.0f / 32768.0f));
  }
}
// Reads `n16` 16-byte vectors with the L2 evict_last policy -- the policy the FFN kernels load their operands with.
// A sweep of twice the L2 size therefore pushes out whatever the previous execution left there, including lines
// that a plain (evict_normal) sweep would never displace.  The sum goes to `sink` so the loads are not dead.
__global__ void __launch_bounds__(256) l2_flush_kernel(const uint4* __restrict__ p, size_t n16, uint32_t* __restrict__ sink) {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  uint32_t acc = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) {
    uint4 v;
    asm volatile("ld.global.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p + i), "l"(pol));
    acc ^= v.x ^ v.y ^ v.z ^ v.w;
  }
  if (acc == 0x9e3779b9u) *sink = acc;     // practically never: keeps the loads alive without a store per thread
}
__global__ void fill_ones_kernel(float* p, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 1.0f;
}
}  // namespace
}  // namespace vibe

namespace vibe {
namespace {
// The sweep itself.  Per point: upload the offsets, max(warmup, 1) untimed calls of run(), then `iters` timed
// executions, median.  The timed executions replay ONE call captured into a CUDA graph, so that an event pair
// brackets the kernels of the call and not the host's work between two launches (tensor-map look-ups, two
// launches with 640 bytes of parameters: ~6 us, more than a lone small expert takes on the device).  Everything
// runs on a stream of the sweep's own, after the caller's stream has drained: the legacy default stream cannot be
// captured.  If the capture fails the calls are timed one by one as launched.
// Every timed execution starts COLD: before its first event an evict_last read sweep of kProfileFlushBytes (twice the
// 126 MB L2) runs on the same stream, outside the event pair.  Without it a sweep point whose operands fit the L2
// (a lone C3 expert: 88 MB of weights; the C2 shape: 9 MB per expert) would be replayed on L2-resident weights and
// read faster than it ever does inside a model, where the other layers' traffic has evicted them.
template <class Run>
vibe_status profile_sweep(int E_loc, const int32_t* tokens_per_expert, int n_points, int mode, int warmup, int iters,
                          float* latency_us, float* samples_us, int32_t* offsets, void* flush, cudaStream_t caller, Run run,
                          int seg_align = 1, void* ffn_ws = nullptr) {
  // ffn_ws: the FFN's split-K / scheduler counters are zeroed AHEAD of every execution, outside the timed region (as
  // the layer entries do before the route kernel); the timed graph holds the two FFN kernels only
  auto pre = [&](cudaStream_t ps) { return ffn_ws ? grouped_ffn_zero_counters(ffn_ws, ps) : VIBE_OK; };
  VIBE_CUDA(cudaStreamSynchronize(caller));
  cudaStream_t st = nullptr;
  VIBE_CUDA(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
  std::vector<cudaEvent_t> ev(2 * (size_t)iters, nullptr);
  vibe_status rc = VIBE_OK;
  for (auto& e : ev)
    if (cudaEventCreate(&e) != cudaSuccess) rc = VIBE_ERR_CUDA;
  if (rc != VIBE_OK) set_error("vibe_profile_expert_latency: cudaEventCreate failed");
  std::vector<int32_t> off(E_loc + 1);
  std::vector<float> t(iters);
  for (int p = 0; p < n_points && rc == VIBE_OK; ++p) {
    const int n = tokens_per_expert[p];
    off[0] = 0;
    // (seg_align > 1: segments start on multiples of it and are that long -- what vibe_permute with that align produces)
    for (int e = 0; e < E_loc; ++e) off[e + 1] = off[e] + ((mode == 0 || e == 0) ? (n + seg_align - 1) / seg_align * seg_align : 0);
    cudaError_t ce = cudaMemcpyAsync(offsets, off.data(), off.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) {
      set_error("vibe_profile_expert_latency: offsets upload failed: %s", cudaGetErrorString(ce));
      rc = VIBE_ERR_CUDA;
      break;
    }
    for (int i = 0; i < std::max(warmup, 1) && rc == VIBE_OK; ++i) {
      rc = pre(st);
      if (rc == VIBE_OK) rc = run(st);
    }
    if (rc == VIBE_OK) rc = pre(st);
    if (rc != VIBE_OK) break;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const vibe_status cs = run(st);
      if (cudaStreamEndCapture(st, &graph) != cudaSuccess || cs != VIBE_OK) {
        if (graph) cudaGraphDestroy(graph);
        graph = nullptr;
      }
      if (graph && cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
    }
    (void)cudaGetLastError();      // a failed capture leaves a sticky-free error behind; the fallback below still works
    for (int i = 0; i < iters && rc == VIBE_OK; ++i) {
      rc = pre(st);
      if (rc != VIBE_OK) break;
      l2_flush_kernel<<<num_sms() * 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(flush), kProfileFlushBytes / 16,
                                                     reinterpret_cast<uint32_t*>(flush));
      count_launch();
      cudaEventRecord(ev[2 * i], st);
      if (exec) {
        if (cudaGraphLaunch(exec, st) != cudaSuccess) {
          set_error("vibe_profile_expert_latency: cudaGraphLaunch failed");
          rc = VIBE_ERR_CUDA;
        }
      } else {
        rc = run(st);
      }
      cudaEventRecord(ev[2 * i + 1], st);
    }
    ce = cudaStreamSynchronize(st);
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
    if (rc != VIBE_OK) break;
    if (ce != cudaSuccess) {
      set_error("vibe_profile_expert_latency: kernel failed: %s", cudaGetErrorString(ce));
      rc = VIBE_ERR_CUDA;
      break;
    }
    for (int i = 0; i < iters; ++i) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ev[2 * i], ev[2 * i + 1]);
      t[i] = ms * 1000.0f;
      if (samples_us) samples_us[(size_t)p * iters + i] = t[i];
    }
    std::sort(t.begin(), t.end());
    const float med = (iters & 1) ? t[iters / 2] : 0.5f * (t[iters / 2 - 1] + t[iters / 2]);
    latency_us[p] = (mode == 0) ? med / (float)E_loc : med;
  }
  for (auto& e : ev)
    if (e) cudaEventDestroy(e);
  cudaStreamDestroy(st);
  return rc;
}
}  // namespace
}  // namespace vibe

extern "C" vibe_status vibe_profile_expert_latency(int32_t E_loc, int32_t d, int32_t f, const void* W1,
                                                   const void* W3, const void* W2,
                                                   const int32_t* tokens_per_expert, int32_t n_points, int32_t mode,
                                                   int32_t warmup, int32_t iters, float* latency_us,
                                                   float* samples_us, void* ws, size_t ws_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(tokens_per_expert && latency_us && n_points >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency: need tokens_per_expert, latency_us, n_points >= 1");
  VIBE_REQUIRE(mode == 0 || mode == 1, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency: mode must be 0 or 1");
  VIBE_REQUIRE(warmup >= 0 && iters >= 1 && iters <= 100000, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency: need warmup >= 0, 1 <= iters <= 100000");
  int n_max = 0;
  for (int p = 0; p < n_points; ++p) {
    VIBE_REQUIRE(tokens_per_expert[p] >= 0, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency: negative token count");
    n_max = std::max(n_max, tokens_per_expert[p]);
  }
  VIBE_REQUIRE((int64_t)E_loc * std::max(n_max, 1) < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency: E_loc * max tokens >= 2^31");
  const int R_cap = E_loc * std::max(n_max, 1);
  const size_t need = vibe_workspace_bytes(VIBE_WS_PROFILE, n_max, 1, E_loc, E_loc, d, f, 1);
  VIBE_REQUIRE(ws != nullptr && ws_bytes >= need && (reinterpret_cast<uintptr_t>(ws) & 255u) == 0, VIBE_ERR_WORKSPACE,
               "vibe_profile_expert_latency: workspace needs %zu bytes, 256-byte aligned (got %zu)", need, ws_bytes);
  char* base = reinterpret_cast<char*>(ws);
  void* Xp = base;
  void* Y = base + round_up((size_t)R_cap * d * 2, 256);
  void* H = base + 2 * round_up((size_t)R_cap * d * 2, 256);
  int32_t* offsets = reinterpret_cast<int32_t*>(base + 2 * round_up((size_t)R_cap * d * 2, 256) +
                                                round_up((size_t)R_cap * f * 2, 256));
  void* flush = base + need - kProfileFlushBytes;
  void* ffn_ws = base + need - kProfileFlushBytes - round_up(grouped_ffn_ws_bytes(), 256);
  vibe_status s = grouped_ffn_check(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H, Y);
  if (s != VIBE_OK) return s;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  fill_pattern_kernel<<<num_sms() * 4, 256, 0, st>>>(reinterpret_cast<__nv_bfloat16*>(Xp), (size_t)R_cap * d);
  VIBE_LAUNCH_CHECK("fill_pattern_kernel");

  VIBE_CUDA(cudaMemsetAsync(flush, 0, kProfileFlushBytes, st));
  return profile_sweep(E_loc, tokens_per_expert, n_points, mode, warmup, iters, latency_us, samples_us, offsets, flush, st,
                       [&](cudaStream_t ps) {
                         return grouped_ffn_impl(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H, Y, ps, nullptr, nullptr, ffn_ws,
                                                 grouped_ffn_ws_bytes(), true);
                       },
                       1, ffn_ws);
}

extern "C" vibe_status vibe_profile_expert_latency_fp8(int32_t E_loc, int32_t d, int32_t f, const void* W1q,
                                                       const float* s1, const void* W3q, const float* s3,
                                                       const void* W2q, const float* s2, const float* h_scale,
                                                       const int32_t* tokens_per_expert, int32_t n_points,
                                                       int32_t mode, int32_t warmup, int32_t iters, float* latency_us,
                                                       float* samples_us, void* ws, size_t ws_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(tokens_per_expert && latency_us && n_points >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_fp8: need tokens_per_expert, latency_us, n_points >= 1");
  VIBE_REQUIRE(mode == 0 || mode == 1, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency_fp8: mode must be 0 or 1");
  VIBE_REQUIRE(warmup >= 0 && iters >= 1 && iters <= 100000, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_fp8: need warmup >= 0, 1 <= iters <= 100000");
  VIBE_REQUIRE(W1q && s1 && W3q && s3 && W2q && s2 && h_scale, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_fp8: NULL weights / scales");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0 && E_loc >= 1, VIBE_ERR_UNSUPPORTED,
               "vibe_profile_expert_latency_fp8: d and f must be multiples of 128");
  int n_max = 0;
  for (int p = 0; p < n_points; ++p) {
    VIBE_REQUIRE(tokens_per_expert[p] >= 0, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency_fp8: negative token count");
    n_max = std::max(n_max, tokens_per_expert[p]);
  }
  VIBE_REQUIRE((int64_t)E_loc * std::max(n_max, 1) < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_fp8: E_loc * max tokens >= 2^31");
  const int R_cap = E_loc * std::max(n_max, 1);
  const size_t base_need = round_up(vibe_workspace_bytes(VIBE_WS_PROFILE, n_max, 1, E_loc, E_loc, d, f, 1), 256);
  const size_t need = base_need + round_up((size_t)R_cap * 4, 256);
  VIBE_REQUIRE(ws != nullptr && ws_bytes >= need && (reinterpret_cast<uintptr_t>(ws) & 255u) == 0, VIBE_ERR_WORKSPACE,
               "vibe_profile_expert_latency_fp8: workspace needs %zu bytes, 256-byte aligned (got %zu)", need, ws_bytes);
  // the bf16 profile's workspace layout with one-byte activations (Xq | Y | Hq | offsets), row scales appended
  char* base = reinterpret_cast<char*>(ws);
  void* Xq = base;
  void* Y = base + round_up((size_t)R_cap * d * 2, 256);
  char* Hreg = base + 2 * round_up((size_t)R_cap * d * 2, 256);
  void* Hq = Hreg;
  int32_t* offsets = reinterpret_cast<int32_t*>(Hreg + round_up((size_t)R_cap * f * 2, 256));
  float* row_scale = reinterpret_cast<float*>(base + base_need);
  void* flush = base + base_need - kProfileFlushBytes;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // arbitrary finite codes (0x38 = 1.0) and unit row scales: latency does not depend on the values
  VIBE_CUDA(cudaMemsetAsync(Xq, 0x38, (size_t)R_cap * d, st));
  fill_ones_kernel<<<num_sms() * 2, 256, 0, st>>>(row_scale, (size_t)R_cap);
  VIBE_LAUNCH_CHECK("fill_ones_kernel");
  VIBE_CUDA(cudaMemsetAsync(flush, 0, kProfileFlushBytes, st));
  return profile_sweep(E_loc, tokens_per_expert, n_points, mode, warmup, iters, latency_us, samples_us, offsets, flush, st, [&](cudaStream_t ps) {
    return grouped_ffn_fp8_impl(Xq, row_scale, offsets, E_loc, R_cap, d, f, W1q, s1, W3q, s3, W2q, s2, h_scale, Hq, Y, ps);
  });
}

extern "C" vibe_status vibe_profile_expert_latency_mxfp8(int32_t E_loc, int32_t d, int32_t f, const void* W1q,
                                                         const void* W3q, const void* sf13, const void* W2q,
                                                         const void* sf2, const int32_t* tokens_per_expert,
                                                         int32_t n_points, int32_t mode, int32_t warmup, int32_t iters,
                                                         float* latency_us, float* samples_us, void* ws, size_t ws_bytes,
                                                         void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(tokens_per_expert && latency_us && n_points >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_mxfp8: need tokens_per_expert, latency_us, n_points >= 1");
  VIBE_REQUIRE(mode == 0 || mode == 1, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency_mxfp8: mode must be 0 or 1");
  VIBE_REQUIRE(warmup >= 0 && iters >= 1 && iters <= 100000, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_mxfp8: need warmup >= 0, 1 <= iters <= 100000");
  VIBE_REQUIRE(W1q && W3q && sf13 && W2q && sf2, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency_mxfp8: NULL weights / scales");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0 && E_loc >= 1 && E_loc <= 512, VIBE_ERR_UNSUPPORTED,
               "vibe_profile_expert_latency_mxfp8: d and f must be multiples of 128, E_loc <= 512");
  int n_max = 0;
  for (int p = 0; p < n_points; ++p) {
    VIBE_REQUIRE(tokens_per_expert[p] >= 0, VIBE_ERR_INVALID_ARG, "vibe_profile_expert_latency_mxfp8: negative token count");
    n_max = std::max(n_max, tokens_per_expert[p]);
  }
  const int n_pad = std::max((n_max + kMxRowAlign - 1) / kMxRowAlign * kMxRowAlign, kMxRowAlign);
  VIBE_REQUIRE((int64_t)E_loc * n_pad < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG,
               "vibe_profile_expert_latency_mxfp8: E_loc * max tokens >= 2^31");
  const int R_cap = E_loc * n_pad;
  const size_t base_need = round_up(vibe_workspace_bytes(VIBE_WS_PROFILE, n_pad, 1, E_loc, E_loc, d, f, 1), 256);
  const size_t xsf_b = round_up(vibe_mxfp8_sf_bytes(VIBE_MX_SF_TOKENS, R_cap, d, 1), 256);
  const size_t hsf_b = round_up(vibe_mxfp8_sf_bytes(VIBE_MX_SF_TOKENS, R_cap, f, 1), 256);
  const size_t need = base_need + xsf_b + hsf_b;
  VIBE_REQUIRE(ws != nullptr && ws_bytes >= need && (reinterpret_cast<uintptr_t>(ws) & 255u) == 0, VIBE_ERR_WORKSPACE,
               "vibe_profile_expert_latency_mxfp8: workspace needs %zu bytes, 256-byte aligned (got %zu)", need, ws_bytes);
  // the bf16 profile's workspace layout with one-byte activations (Xq | Y | Hq | offsets | FFN ws | flush), scales appended
  char* base = reinterpret_cast<char*>(ws);
  void* Xq = base;
  void* Y = base + round_up((size_t)R_cap * d * 2, 256);
  char* Hreg = base + 2 * round_up((size_t)R_cap * d * 2, 256);
  void* Hq = Hreg;
  int32_t* offsets = reinterpret_cast<int32_t*>(Hreg + round_up((size_t)R_cap * f * 2, 256));
  void* flush = base + base_need - kProfileFlushBytes;
  void* ffn_ws = base + base_need - kProfileFlushBytes - round_up(grouped_ffn_ws_bytes(), 256);
  void* xsf = base + base_need;
  void* hsf = base + base_need + xsf_b;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // arbitrary finite codes (0x38 = 1.0) and unit scales (byte 127): latency does not depend on the values
  VIBE_CUDA(cudaMemsetAsync(Xq, 0x38, (size_t)R_cap * d, st));
  VIBE_CUDA(cudaMemsetAsync(xsf, 127, xsf_b, st));
  VIBE_CUDA(cudaMemsetAsync(hsf, 127, hsf_b, st));
  VIBE_CUDA(cudaMemsetAsync(flush, 0, kProfileFlushBytes, st));
  return profile_sweep(E_loc, tokens_per_expert, n_points, mode, warmup, iters, latency_us, samples_us, offsets, flush, st,
                       [&](cudaStream_t ps) {
                         return grouped_ffn_mxfp8_impl(Xq, xsf, offsets, E_loc, R_cap, d, f, W1q, W3q, sf13, W2q, sf2, Hq, hsf, Y, ps,
                                                       ffn_ws, grouped_ffn_ws_bytes(), true);
                       },
                       kMxRowAlign, ffn_ws);
}

// Measurement utility: evict the L2 (evict_last read sweep, see l2_flush_kernel) before a timed region.
extern "C" vibe_status vibe_l2_flush(void* scratch, size_t bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(scratch != nullptr && bytes >= 64 && aligned16(scratch), VIBE_ERR_INVALID_ARG,
               "vibe_l2_flush: scratch must be a 16-byte aligned device buffer of at least 64 bytes");
  l2_flush_kernel<<<num_sms() * 8, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(
      reinterpret_cast<const uint4*>(scratch), bytes / 16, reinterpret_cast<uint32_t*>(scratch));
  VIBE_LAUNCH_CHECK("l2_flush_kernel");
  return VIBE_OK;
}
