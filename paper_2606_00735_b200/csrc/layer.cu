// layer.cu -- the whole per-GPU MoE layer (a1..a5) as one enqueue, from device or host buffers.
#include "common.cuh"

#include <cmath>
#include <mutex>


extern "C" vibe_status vibe_moe_layer_forward(const vibe_route_cfg* cfg, const float* logits, const void* X,
                                              const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                              int32_t E_loc, const void* W1, const void* W3, const void* W2,
                                              void* out, int32_t* counts, int32_t* topk_ids, float* topk_w,
                                              void* arena, size_t arena_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward: cfg is NULL");
  VIBE_REQUIRE(T >= 0 && d >= 8 && f >= 8 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward: bad sizes");
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward: need 1 <= k <= E");
  {
    vibe_status lim = grouped_ffn_limits("vibe_moe_layer_forward", E_loc, d, f, W1, W3, W2);   // before any launch
    if (lim != VIBE_OK) return lim;
  }
  VIBE_REQUIRE(out != nullptr && counts != nullptr && logits != nullptr && (T == 0 || X != nullptr), VIBE_ERR_INVALID_ARG,
               "vibe_moe_layer_forward: NULL tensor");
  const LayerArena a = layer_arena(T, k, E_loc, d, f);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= a.total && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward: arena needs %zu bytes, 256-byte aligned (got %zu)", a.total,
               arena_bytes);
  VIBE_REQUIRE(a.R_cap < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward: row capacity >= 2^31");
  char* base = reinterpret_cast<char*>(arena);
  int32_t* ids = topk_ids ? topk_ids : reinterpret_cast<int32_t*>(base + a.ids);
  float* w = topk_w ? topk_w : reinterpret_cast<float*>(base + a.w);
  int32_t* offsets = reinterpret_cast<int32_t*>(base + a.offsets);
  int32_t* r2a = reinterpret_cast<int32_t*>(base + a.r2a);
  int32_t* a2r = reinterpret_cast<int32_t*>(base + a.a2r);
  void* Xp = base + a.Xp;
  void* H = base + a.H;
  void* Y = base + a.Y;
  vibe_status s;
  // the split-K counters of the FFN are zeroed HERE, ahead of the route kernel: a memset between the permutation and
  // the FFN kernels would cut their programmatic-dependent-launch chain
  if (T > 0 && (s = grouped_ffn_zero_counters(base + a.ffn_ws, reinterpret_cast<cudaStream_t>(stream))) != VIBE_OK) return s;
  if ((s = vibe_route_topk(cfg, logits, T, ids, w, counts, stream)) != VIBE_OK) return s;
  if ((s = vibe_permute(X, ids, counts, expert_map, T, d, k, E, E_loc, 1, Xp, offsets, r2a, a2r, base + a.perm_ws,
                        permute_ws_bytes(T, k, E_loc), stream)) != VIBE_OK)
    return s;
  if (T == 0) return VIBE_OK;
  if ((s = grouped_ffn_check(Xp, offsets, E_loc, (int)a.R_cap, d, f, W1, W3, W2, H, Y)) != VIBE_OK) return s;
  if ((s = grouped_ffn_impl(Xp, offsets, E_loc, (int)a.R_cap, d, f, W1, W3, W2, H, Y, reinterpret_cast<cudaStream_t>(stream),
                            nullptr, nullptr, base + a.ffn_ws, grouped_ffn_ws_bytes(), true)) != VIBE_OK)
    return s;
  return vibe_combine(Y, a2r, w, T, k, d, out, stream);
}

namespace {

constexpr int kMaxHostChunks = 8;

// Two copy streams and the events that order them against the caller's stream; created once per device.
constexpr int kMaxTickets = 8;     // outstanding asynchronous host calls per device

struct HostPipe {
  cudaStream_t in = nullptr, out = nullptr;
  cudaEvent_t entry = nullptr, out_done = nullptr;
  cudaEvent_t in_done[kMaxHostChunks] = {}, comp_done[kMaxHostChunks] = {};
  // the asynchronous entry: one event triple per ticket slot
  cudaEvent_t t_entry[kMaxTickets] = {}, t_in[kMaxTickets] = {}, t_comp[kMaxTickets] = {}, t_done[kMaxTickets] = {};
  bool t_busy[kMaxTickets] = {};
  bool ready = false;
  std::mutex in_use;   // one pipelined call per device at a time (the events are per device, and the call waits anyway)
};

vibe_status host_pipe(HostPipe** pp) {
  static std::mutex mu;
  static HostPipe pipes[64];
  int dev = 0;
  VIBE_CUDA(cudaGetDevice(&dev));
  VIBE_REQUIRE(dev >= 0 && dev < 64, VIBE_ERR_CUDA, "vibe_moe_layer_forward_host: device ordinal %d", dev);
  std::lock_guard<std::mutex> lock(mu);
  HostPipe& hp = pipes[dev];
  if (!hp.ready) {
    VIBE_CUDA(cudaStreamCreateWithFlags(&hp.in, cudaStreamNonBlocking));
    VIBE_CUDA(cudaStreamCreateWithFlags(&hp.out, cudaStreamNonBlocking));
    VIBE_CUDA(cudaEventCreateWithFlags(&hp.entry, cudaEventDisableTiming));
    VIBE_CUDA(cudaEventCreateWithFlags(&hp.out_done, cudaEventDisableTiming));
    for (int c = 0; c < kMaxHostChunks; ++c) {
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.in_done[c], cudaEventDisableTiming));
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.comp_done[c], cudaEventDisableTiming));
    }
    for (int c = 0; c < kMaxTickets; ++c) {
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.t_entry[c], cudaEventDisableTiming));
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.t_in[c], cudaEventDisableTiming));
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.t_comp[c], cudaEventDisableTiming));
      VIBE_CUDA(cudaEventCreateWithFlags(&hp.t_done[c], cudaEventDisableTiming));
    }
    hp.ready = true;
  }
  *pp = &hp;
  return VIBE_OK;
}

__global__ void sum_count_parts_kernel(const int32_t* __restrict__ parts, int n_parts, int E, int32_t* __restrict__ counts) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  int32_t c = 0;
  for (int p = 0; p < n_parts; ++p) c += parts[(size_t)p * E + e];
  counts[e] = c;
}

// Number of token chunks that minimises a three-stage (copy in, compute, copy out) pipeline estimate:
// makespan = a + b + c + (C - 1) * max(a, b, c) for per-chunk stage times a, b, c.  The compute estimate is the
// larger of the FFN's flop time (with an efficiency that falls off below ~128 rows per expert tile) and its weight
// streaming time; the constants are round B200 / PCIe Gen5 figures -- only the ordering of the candidates matters.
int auto_host_chunks(int T, int k, int E, int E_loc, int d, int f) {
  const double pcie = 50e9, hbm = 6.0e12, tensor = 1.25e15, launch = 40e-6;
  const double in_bytes = (double)T * E * 4 + (double)T * d * 2, out_bytes = (double)T * d * 2;
  int best = 1;
  double best_t = 0;
  for (int C = 1; C <= kMaxHostChunks; ++C) {
    const double Tc = (double)T / C;
    if (C > 1 && Tc < 256) break;
    const double n = Tc * k / E;  // mean rows per expert in one chunk
    const double flops = 6.0 * Tc * k * d * f * ((double)E_loc / E);
    const double b = fmax(flops / (tensor * n / (n + 128.0)), 6.0 * d * f * E_loc / hbm) + launch;
    const double a = in_bytes / C / pcie, c = out_bytes / C / pcie;
    const double t = a + b + c + (C - 1) * fmax(a, fmax(b, c));
    if (C == 1 || t < best_t) best = C, best_t = t;
  }
  return best;
}

}  // namespace

extern "C" vibe_status vibe_moe_layer_forward_host_chunked(const vibe_route_cfg* cfg, const float* logits_h,
                                                           const void* X_h, const int32_t* expert_map, int32_t T,
                                                           int32_t d, int32_t f, int32_t E_loc, const void* W1,
                                                           const void* W3, const void* W2, void* out_h,
                                                           int32_t* counts_h, int32_t n_chunks, void* arena,
                                                           size_t arena_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: cfg is NULL");
  VIBE_REQUIRE(T >= 1 && d >= 8 && f >= 8 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: bad sizes");
  VIBE_REQUIRE(logits_h && X_h && out_h && counts_h, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: NULL host buffer");
  VIBE_REQUIRE(n_chunks >= 0 && n_chunks <= kMaxHostChunks, VIBE_ERR_INVALID_ARG,
               "vibe_moe_layer_forward_host: n_chunks must be 0 (choose) .. %d", kMaxHostChunks);
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: need 1 <= k <= E");
  {
    vibe_status lim = grouped_ffn_limits("vibe_moe_layer_forward_host", E_loc, d, f, W1, W3, W2);   // before any copy / launch
    if (lim != VIBE_OK) return lim;
  }
  const size_t inner = vibe_workspace_bytes(VIBE_WS_LAYER, T, k, E, E_loc, d, f, 1);
  const size_t need = vibe_workspace_bytes(VIBE_WS_LAYER_HOST, T, k, E, E_loc, d, f, 1);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= need && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward_host: arena needs %zu bytes, 256-byte aligned (got %zu)",
               need, arena_bytes);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  char* p = reinterpret_cast<char*>(arena) + inner;
  float* logits_d = reinterpret_cast<float*>(p);
  p += round_up((size_t)T * E * 4, 256);
  char* X_d = p;
  p += round_up((size_t)T * d * 2, 256);
  char* out_d = p;
  p += round_up((size_t)T * d * 2, 256);
  int32_t* counts_d = reinterpret_cast<int32_t*>(p);
  p += round_up((size_t)E * 4, 256);
  int32_t* count_parts = reinterpret_cast<int32_t*>(p);

  // chunks of Tc tokens (a multiple of 16, so that every chunk of every buffer starts 64-byte aligned)
  int C = n_chunks ? n_chunks : auto_host_chunks(T, k, E, E_loc, d, f);
  int Tc = (int)round_up((size_t)(T + C - 1) / C, 16);
  C = (T + Tc - 1) / Tc;
  const char* Xh = reinterpret_cast<const char*>(X_h);
  char* outh = reinterpret_cast<char*>(out_h);
  if (C == 1) {
    VIBE_CUDA(cudaMemcpyAsync(logits_d, logits_h, (size_t)T * E * 4, cudaMemcpyHostToDevice, st));
    VIBE_CUDA(cudaMemcpyAsync(X_d, X_h, (size_t)T * d * 2, cudaMemcpyHostToDevice, st));
    vibe_status s = vibe_moe_layer_forward(cfg, logits_d, X_d, expert_map, T, d, f, E_loc, W1, W3, W2, out_d, counts_d,
                                           nullptr, nullptr, arena, inner, stream);
    if (s != VIBE_OK) return s;
    VIBE_CUDA(cudaMemcpyAsync(out_h, out_d, (size_t)T * d * 2, cudaMemcpyDeviceToHost, st));
    VIBE_CUDA(cudaMemcpyAsync(counts_h, counts_d, (size_t)E * 4, cudaMemcpyDeviceToHost, st));
    VIBE_CUDA(cudaStreamSynchronize(st));
    return VIBE_OK;
  }
  // Chunk c's copy-in (stream `in`), layer (caller's stream) and copy-out (stream `out`) overlap with the other
  // chunks' stages; the layer's working buffers are shared by the chunks, which run in order on the caller's stream.
  HostPipe* hp = nullptr;
  vibe_status s = host_pipe(&hp);
  if (s != VIBE_OK) return s;
  std::lock_guard<std::mutex> one_call(hp->in_use);
  VIBE_CUDA(cudaEventRecord(hp->entry, st));
  VIBE_CUDA(cudaStreamWaitEvent(hp->in, hp->entry, 0));
  VIBE_CUDA(cudaStreamWaitEvent(hp->out, hp->entry, 0));
  for (int c = 0; c < C; ++c) {
    const int t0 = c * Tc, tn = (T - t0 < Tc) ? T - t0 : Tc;
    VIBE_CUDA(cudaMemcpyAsync(logits_d + (size_t)t0 * E, logits_h + (size_t)t0 * E, (size_t)tn * E * 4,
                              cudaMemcpyHostToDevice, hp->in));
    VIBE_CUDA(cudaMemcpyAsync(X_d + (size_t)t0 * d * 2, Xh + (size_t)t0 * d * 2, (size_t)tn * d * 2,
                              cudaMemcpyHostToDevice, hp->in));
    VIBE_CUDA(cudaEventRecord(hp->in_done[c], hp->in));
    VIBE_CUDA(cudaStreamWaitEvent(st, hp->in_done[c], 0));
    s = vibe_moe_layer_forward(cfg, logits_d + (size_t)t0 * E, X_d + (size_t)t0 * d * 2, expert_map, tn, d, f, E_loc, W1,
                               W3, W2, out_d + (size_t)t0 * d * 2, count_parts + (size_t)c * E, nullptr, nullptr, arena,
                               inner, stream);
    if (s != VIBE_OK) {
      // copies of this and earlier chunks may still be in flight: the host buffers must be quiet when we return
      cudaStreamSynchronize(hp->in);
      cudaStreamSynchronize(st);
      cudaStreamSynchronize(hp->out);
      return s;
    }
    VIBE_CUDA(cudaEventRecord(hp->comp_done[c], st));
    VIBE_CUDA(cudaStreamWaitEvent(hp->out, hp->comp_done[c], 0));
    VIBE_CUDA(cudaMemcpyAsync(outh + (size_t)t0 * d * 2, out_d + (size_t)t0 * d * 2, (size_t)tn * d * 2,
                              cudaMemcpyDeviceToHost, hp->out));
  }
  sum_count_parts_kernel<<<(E + 255) / 256, 256, 0, st>>>(count_parts, C, E, counts_d);
  VIBE_LAUNCH_CHECK("sum_count_parts_kernel");
  VIBE_CUDA(cudaMemcpyAsync(counts_h, counts_d, (size_t)E * 4, cudaMemcpyDeviceToHost, st));
  VIBE_CUDA(cudaEventRecord(hp->out_done, hp->out));
  VIBE_CUDA(cudaStreamWaitEvent(st, hp->out_done, 0));
  VIBE_CUDA(cudaStreamSynchronize(st));
  return VIBE_OK;
}

extern "C" vibe_status vibe_moe_layer_forward_host(const vibe_route_cfg* cfg, const float* logits_h,
                                                   const void* X_h, const int32_t* expert_map, int32_t T, int32_t d,
                                                   int32_t f, int32_t E_loc, const void* W1, const void* W3,
                                                   const void* W2, void* out_h, int32_t* counts_h, void* arena,
                                                   size_t arena_bytes, void* stream) {
  return vibe_moe_layer_forward_host_chunked(cfg, logits_h, X_h, expert_map, T, d, f, E_loc, W1, W3, W2, out_h,
                                             counts_h, 0, arena, arena_bytes, stream);
}

extern "C" vibe_status vibe_moe_layer_forward_host_async(const vibe_route_cfg* cfg, const float* logits_h, const void* X_h,
                                                         const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                                         int32_t E_loc, const void* W1, const void* W3, const void* W2,
                                                         void* out_h, int32_t* counts_h, void* arena, size_t arena_bytes,
                                                         void* stream, int32_t* ticket) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr && ticket != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host_async: cfg / ticket is NULL");
  VIBE_REQUIRE(T >= 1 && d >= 8 && f >= 8 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host_async: bad sizes");
  VIBE_REQUIRE(logits_h && X_h && out_h && counts_h, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host_async: NULL host buffer");
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host_async: need 1 <= k <= E");
  {
    vibe_status lim = grouped_ffn_limits("vibe_moe_layer_forward_host_async", E_loc, d, f, W1, W3, W2);
    if (lim != VIBE_OK) return lim;
  }
  const size_t inner = vibe_workspace_bytes(VIBE_WS_LAYER, T, k, E, E_loc, d, f, 1);
  const size_t need = vibe_workspace_bytes(VIBE_WS_LAYER_HOST, T, k, E, E_loc, d, f, 1);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= need && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward_host_async: arena needs %zu bytes, 256-byte aligned (got %zu)",
               need, arena_bytes);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  char* p = reinterpret_cast<char*>(arena) + inner;
  float* logits_d = reinterpret_cast<float*>(p);
  p += round_up((size_t)T * E * 4, 256);
  char* X_d = p;
  p += round_up((size_t)T * d * 2, 256);
  char* out_d = p;
  p += round_up((size_t)T * d * 2, 256);
  int32_t* counts_d = reinterpret_cast<int32_t*>(p);
  HostPipe* hp = nullptr;
  vibe_status s = host_pipe(&hp);
  if (s != VIBE_OK) return s;
  int dev = current_device(), slot = -1;
  {
    std::lock_guard<std::mutex> lk(hp->in_use);
    for (int c = 0; c < kMaxTickets && slot < 0; ++c)
      if (!hp->t_busy[c]) slot = c;
    VIBE_REQUIRE(slot >= 0, VIBE_ERR_UNSUPPORTED, "vibe_moe_layer_forward_host_async: %d tickets outstanding on this device", kMaxTickets);
    // copy-in (NOT ordered after the work on `stream`: the previous step's kernels are there, and the copy must
    // overlap them; the host inputs are the host's and ready when the call is made, the arena is free by contract),
    // then the layer on `stream`, then the copy-out; the three queues of consecutive calls overlap
    VIBE_CUDA(cudaMemcpyAsync(logits_d, logits_h, (size_t)T * E * 4, cudaMemcpyHostToDevice, hp->in));
    VIBE_CUDA(cudaMemcpyAsync(X_d, X_h, (size_t)T * d * 2, cudaMemcpyHostToDevice, hp->in));
    VIBE_CUDA(cudaEventRecord(hp->t_in[slot], hp->in));
    VIBE_CUDA(cudaStreamWaitEvent(st, hp->t_in[slot], 0));
    s = vibe_moe_layer_forward(cfg, logits_d, X_d, expert_map, T, d, f, E_loc, W1, W3, W2, out_d, counts_d, nullptr, nullptr,
                               arena, inner, stream);
    if (s != VIBE_OK) {
      cudaStreamSynchronize(hp->in);
      cudaStreamSynchronize(st);
      return s;
    }
    VIBE_CUDA(cudaEventRecord(hp->t_comp[slot], st));
    VIBE_CUDA(cudaStreamWaitEvent(hp->out, hp->t_comp[slot], 0));
    VIBE_CUDA(cudaMemcpyAsync(out_h, out_d, (size_t)T * d * 2, cudaMemcpyDeviceToHost, hp->out));
    VIBE_CUDA(cudaMemcpyAsync(counts_h, counts_d, (size_t)E * 4, cudaMemcpyDeviceToHost, hp->out));
    VIBE_CUDA(cudaEventRecord(hp->t_done[slot], hp->out));
    hp->t_busy[slot] = true;
  }
  *ticket = dev * kMaxTickets + slot;
  return VIBE_OK;
}

extern "C" vibe_status vibe_host_wait(int32_t ticket) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(ticket >= 0 && ticket < kMaxDevices * kMaxTickets, VIBE_ERR_INVALID_ARG, "vibe_host_wait: bad ticket %d", ticket);
  const int dev = ticket / kMaxTickets, slot = ticket % kMaxTickets;
  int cur = 0;
  VIBE_CUDA(cudaGetDevice(&cur));
  HostPipe* hp = nullptr;
  if (cur != dev) VIBE_CUDA(cudaSetDevice(dev));
  vibe_status s = host_pipe(&hp);
  if (s == VIBE_OK) {
    bool busy;
    {
      std::lock_guard<std::mutex> lk(hp->in_use);
      busy = hp->t_busy[slot];
    }
    if (!busy) {
      set_error("vibe_host_wait: ticket %d is not outstanding", ticket);
      s = VIBE_ERR_INVALID_ARG;
    } else {
      const cudaError_t e = cudaEventSynchronize(hp->t_done[slot]);
      std::lock_guard<std::mutex> lk(hp->in_use);
      hp->t_busy[slot] = false;
      if (e != cudaSuccess) {
        set_error("vibe_host_wait: %s", cudaGetErrorString(e));
        s = VIBE_ERR_CUDA;
      }
    }
  }
  if (cur != dev) cudaSetDevice(cur);
  return s;
}

extern "C" vibe_status vibe_moe_layer_forward_fp8(const vibe_route_cfg* cfg, const float* logits, const void* X,
                                                  const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                                  int32_t E_loc, const void* W1q, const float* s1, const void* W3q,
                                                  const float* s3, const void* W2q, const float* s2,
                                                  const float* h_scale, void* out, int32_t* counts, void* arena,
                                                  size_t arena_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: cfg is NULL");
  VIBE_REQUIRE(T >= 0 && d >= 128 && f >= 128 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: bad sizes");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_moe_layer_forward_fp8: d and f must be multiples of 128 (d=%d f=%d)", d, f);
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: need 1 <= k <= E");
  VIBE_REQUIRE(E_loc <= 512, VIBE_ERR_UNSUPPORTED, "vibe_moe_layer_forward_fp8: E_loc > 512 not implemented");
  VIBE_REQUIRE(W1q && s1 && W3q && s3 && W2q && s2 && h_scale && aligned16(W1q) && aligned16(W3q) && aligned16(W2q) && out &&
                   counts && logits,
               VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: NULL or misaligned tensor");
  const LayerArenaFp8 a = layer_arena_fp8(T, k, E_loc, d, f);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= a.total && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward_fp8: arena needs %zu bytes, 256-byte aligned (got %zu)",
               a.total, arena_bytes);
  VIBE_REQUIRE(a.R_cap < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: row capacity >= 2^31");
  char* base = reinterpret_cast<char*>(arena);
  int32_t* ids = reinterpret_cast<int32_t*>(base + a.ids);
  float* w = reinterpret_cast<float*>(base + a.w);
  int32_t* offsets = reinterpret_cast<int32_t*>(base + a.offsets);
  int32_t* r2a = reinterpret_cast<int32_t*>(base + a.r2a);
  int32_t* a2r = reinterpret_cast<int32_t*>(base + a.a2r);
  float* tok_scale = reinterpret_cast<float*>(base + a.tok_scale);
  float* row_scale = reinterpret_cast<float*>(base + a.row_scale);
  vibe_status s;
  if (T > 0 && (s = grouped_ffn_zero_counters(base + a.ffn_ws, reinterpret_cast<cudaStream_t>(stream))) != VIBE_OK) return s;
  if ((s = vibe_route_topk(cfg, logits, T, ids, w, counts, stream)) != VIBE_OK) return s;
  // tokens are quantised BEFORE the permutation (T rows instead of T*k), and the permutation then moves
  // one-byte elements: to vibe_permute an e4m3 row of d bytes is a bf16 row of d/2 elements
  // (on an expert-parallel shard only the tokens with a resident expert are quantised)
  VIBE_REQUIRE(T == 0 || (X != nullptr && aligned16(X)), VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_fp8: X NULL or misaligned");
  if ((s = fp8_quantize_resident_tokens(X, T, d, base + a.Xq, tok_scale, (expert_map && E_loc < E) ? ids : nullptr,
                                        expert_map, k, E, E_loc, reinterpret_cast<cudaStream_t>(stream))) != VIBE_OK)
    return s;
  if ((s = vibe_permute(base + a.Xq, ids, counts, expert_map, T, d / 2, k, E, E_loc, 1, base + a.Xpq, offsets, r2a, a2r,
                        base + a.perm_ws, permute_ws_bytes(T, k, E_loc), stream)) != VIBE_OK)
    return s;
  if (T == 0) return VIBE_OK;
  if ((s = fp8_gather_row_scales(tok_scale, r2a, offsets, E_loc, k, (int)a.R_cap, row_scale,
                                 reinterpret_cast<cudaStream_t>(stream))) != VIBE_OK)
    return s;
  if ((s = grouped_ffn_fp8_impl(base + a.Xpq, row_scale, offsets, E_loc, (int)a.R_cap, d, f, W1q, s1, W3q, s3, W2q, s2, h_scale,
                                base + a.Hq, base + a.Y, reinterpret_cast<cudaStream_t>(stream), base + a.ffn_ws,
                                grouped_ffn_ws_bytes(), true)) != VIBE_OK)
    return s;
  return vibe_combine(base + a.Y, a2r, w, T, k, d, out, stream);
}

extern "C" vibe_status vibe_moe_layer_forward_mxfp8(const vibe_route_cfg* cfg, const float* logits, const void* X,
                                                    const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                                    int32_t E_loc, const void* W1q, const void* W3q, const void* sf13,
                                                    const void* W2q, const void* sf2, void* out, int32_t* counts,
                                                    void* arena, size_t arena_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: cfg is NULL");
  VIBE_REQUIRE(T >= 0 && d >= 128 && f >= 128 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: bad sizes");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_moe_layer_forward_mxfp8: d and f must be multiples of 128 (d=%d f=%d)", d, f);
  VIBE_REQUIRE(E_loc <= 512, VIBE_ERR_UNSUPPORTED, "vibe_moe_layer_forward_mxfp8: E_loc > 512 not implemented");
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: need 1 <= k <= E");
  VIBE_REQUIRE(W1q && W3q && sf13 && W2q && sf2 && aligned16(W1q) && aligned16(W3q) && aligned16(sf13) && aligned16(W2q) &&
                   aligned16(sf2),
               VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: weight / scale tensor NULL or not 16-byte aligned");
  const LayerArenaMx a = layer_arena_mx(T, k, E_loc, d, f);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= a.total && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward_mxfp8: arena needs %zu bytes, 256-byte aligned (got %zu)",
               a.total, arena_bytes);
  VIBE_REQUIRE(a.R_cap < (int64_t)INT32_MAX, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: row capacity >= 2^31");
  VIBE_REQUIRE(T == 0 || (X != nullptr && aligned16(X)), VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_mxfp8: X NULL or misaligned");
  char* base = reinterpret_cast<char*>(arena);
  int32_t* ids = reinterpret_cast<int32_t*>(base + a.ids);
  float* w = reinterpret_cast<float*>(base + a.w);
  int32_t* offsets = reinterpret_cast<int32_t*>(base + a.offsets);
  int32_t* r2a = reinterpret_cast<int32_t*>(base + a.r2a);
  int32_t* a2r = reinterpret_cast<int32_t*>(base + a.a2r);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  vibe_status s;
  if (T > 0 && (s = grouped_ffn_zero_counters(base + a.ffn_ws, st)) != VIBE_OK) return s;
  if ((s = vibe_route_topk(cfg, logits, T, ids, w, counts, stream)) != VIBE_OK) return s;
  // tokens are quantised BEFORE the permutation (T rows instead of T*k); the permutation then moves one-byte rows
  if ((s = mx_quantize_rows(X, T, d, 32, base + a.Xq, base + a.tok_sf, VIBE_MX_SF_ROWMAJOR, T,
                            (expert_map && E_loc < E) ? ids : nullptr, expert_map, k, E, E_loc, st)) != VIBE_OK)
    return s;
  if ((s = vibe_permute(base + a.Xq, ids, counts, expert_map, T, d / 2, k, E, E_loc, kMxRowAlign, base + a.Xpq, offsets, r2a,
                        a2r, base + a.perm_ws, permute_ws_bytes(T, k, E_loc), stream)) != VIBE_OK)
    return s;
  if (T == 0) return VIBE_OK;
  if ((s = mx_gather_row_sf(base + a.tok_sf, r2a, offsets, E_loc, k, (int)a.R_cap, d, base + a.xsf, st)) != VIBE_OK) return s;
  if ((s = grouped_ffn_mxfp8_impl(base + a.Xpq, base + a.xsf, offsets, E_loc, (int)a.R_cap, d, f, W1q, W3q, sf13, W2q, sf2,
                                  base + a.Hq, base + a.hsf, base + a.Y, st, base + a.ffn_ws, grouped_ffn_ws_bytes(), true)) != VIBE_OK)
    return s;
  return vibe_combine(base + a.Y, a2r, w, T, k, d, out, stream);
}
