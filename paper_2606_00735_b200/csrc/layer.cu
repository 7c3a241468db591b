// layer.cu -- the whole per-GPU MoE layer (a1..a5) as one enqueue, from device or host buffers.
#include "common.cuh"


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
  if ((s = vibe_route_topk(cfg, logits, T, ids, w, counts, stream)) != VIBE_OK) return s;
  if ((s = vibe_permute(X, ids, counts, expert_map, T, d, k, E, E_loc, 1, Xp, offsets, r2a, a2r, base + a.perm_ws,
                        permute_ws_bytes(T, k, E_loc), stream)) != VIBE_OK)
    return s;
  if (T == 0) return VIBE_OK;
  if ((s = vibe_grouped_ffn(Xp, offsets, E_loc, (int32_t)a.R_cap, d, f, W1, W3, W2, H, Y, nullptr, 0, stream)) !=
      VIBE_OK)
    return s;
  return vibe_combine(Y, a2r, w, T, k, d, out, stream);
}

extern "C" vibe_status vibe_moe_layer_forward_host(const vibe_route_cfg* cfg, const float* logits_h,
                                                   const void* X_h, const int32_t* expert_map, int32_t T, int32_t d,
                                                   int32_t f, int32_t E_loc, const void* W1, const void* W3,
                                                   const void* W2, void* out_h, int32_t* counts_h, void* arena,
                                                   size_t arena_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(cfg != nullptr, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: cfg is NULL");
  VIBE_REQUIRE(T >= 1 && d >= 8 && f >= 8 && E_loc >= 1, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: bad sizes");
  VIBE_REQUIRE(logits_h && X_h && out_h && counts_h, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: NULL host buffer");
  const int E = cfg->num_experts, k = cfg->top_k;
  VIBE_REQUIRE(E >= 1 && k >= 1 && k <= E, VIBE_ERR_INVALID_ARG, "vibe_moe_layer_forward_host: need 1 <= k <= E");
  const size_t inner = vibe_workspace_bytes(VIBE_WS_LAYER, T, k, E, E_loc, d, f, 1);
  const size_t need = vibe_workspace_bytes(VIBE_WS_LAYER_HOST, T, k, E, E_loc, d, f, 1);
  VIBE_REQUIRE(arena != nullptr && arena_bytes >= need && (reinterpret_cast<uintptr_t>(arena) & 255u) == 0,
               VIBE_ERR_WORKSPACE, "vibe_moe_layer_forward_host: arena needs %zu bytes, 256-byte aligned (got %zu)",
               need, arena_bytes);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  char* p = reinterpret_cast<char*>(arena) + inner;
  float* logits_d = reinterpret_cast<float*>(p);
  p += round_up((size_t)T * E * 4, 256);
  void* X_d = p;
  p += round_up((size_t)T * d * 2, 256);
  void* out_d = p;
  p += round_up((size_t)T * d * 2, 256);
  int32_t* counts_d = reinterpret_cast<int32_t*>(p);
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
  if ((s = vibe_grouped_ffn_fp8(base + a.Xpq, row_scale, offsets, E_loc, (int32_t)a.R_cap, d, f, W1q, s1, W3q, s3, W2q,
                                s2, h_scale, base + a.Hq, base + a.Y, stream)) != VIBE_OK)
    return s;
  return vibe_combine(base + a.Y, a2r, w, T, k, d, out, stream);
}
