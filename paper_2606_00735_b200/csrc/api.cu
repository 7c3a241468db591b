// api.cu -- status / error text / workspace sizing / launch accounting of libvibe.so.
#include <string.h>
#include <atomic>

#include "common.cuh"

namespace vibe {

static thread_local char g_err[512] = "";
static thread_local long long g_launches = 0;

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
void clear_error() { g_err[0] = '\0'; }
void count_launch(int n) { g_launches += n; }

int current_device() {
  int dev = 0;
  return (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices) ? dev : 0;
}

// SM count of the CURRENT device (cached per device ordinal: a process may drive several GPUs)
int num_sms() {
  static std::atomic<int> sms[kMaxDevices];
  const int dev = current_device();
  int v = sms[dev].load(std::memory_order_relaxed);
  if (v == 0) {
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0)
      sms[dev].store(v, std::memory_order_relaxed);
    else
      return 148;  // B200; only reached when no device is present (launch will fail loudly)
  }
  return v;
}

LayerArena layer_arena(int T, int k, int E_loc, int d, int f) {
  LayerArena a{};
  const size_t A = (size_t)T * k;
  a.R_cap = vibe_rows_cap(T, k, E_loc, 1);
  if (a.R_cap < 1) a.R_cap = 1;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o += round_up(bytes ? bytes : 16, 256);
    return at;
  };
  a.ids = take(A * 4);
  a.w = take(A * 4);
  a.offsets = take((size_t)(E_loc + 1) * 4);
  a.r2a = take((size_t)a.R_cap * 4);
  a.a2r = take(A * 4);
  a.Xp = take((size_t)a.R_cap * d * 2);
  a.H = take((size_t)a.R_cap * f * 2);
  a.Y = take((size_t)a.R_cap * d * 2);
  a.perm_ws = take(permute_ws_bytes(T, k, E_loc));
  a.ffn_ws = take(grouped_ffn_ws_bytes());
  a.total = o;
  return a;
}

LayerArenaFp8 layer_arena_fp8(int T, int k, int E_loc, int d, int f) {
  LayerArenaFp8 a{};
  const size_t A = (size_t)T * k;
  a.R_cap = vibe_rows_cap(T, k, E_loc, 1);
  if (a.R_cap < 1) a.R_cap = 1;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o += round_up(bytes ? bytes : 16, 256);
    return at;
  };
  a.ids = take(A * 4);
  a.w = take(A * 4);
  a.offsets = take((size_t)(E_loc + 1) * 4);
  a.r2a = take((size_t)a.R_cap * 4);
  a.a2r = take(A * 4);
  a.Xq = take((size_t)T * d);
  a.tok_scale = take((size_t)T * 4);
  a.Xpq = take((size_t)a.R_cap * d);
  a.row_scale = take((size_t)a.R_cap * 4);
  a.Hq = take((size_t)a.R_cap * f);
  a.Y = take((size_t)a.R_cap * d * 2);
  a.perm_ws = take(permute_ws_bytes(T, k, E_loc));
  a.ffn_ws = take(grouped_ffn_ws_bytes());
  a.total = o;
  return a;
}

LayerArenaMx layer_arena_mx(int T, int k, int E_loc, int d, int f) {
  LayerArenaMx a{};
  const size_t A = (size_t)T * k;
  a.R_cap = vibe_rows_cap(T, k, E_loc, kMxRowAlign);
  if (a.R_cap < 1) a.R_cap = 1;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o += round_up(bytes ? bytes : 16, 256);
    return at;
  };
  const size_t Rb = (size_t)mx_row_blocks((int)a.R_cap);
  a.ids = take(A * 4);
  a.w = take(A * 4);
  a.offsets = take((size_t)(E_loc + 1) * 4);
  a.r2a = take((size_t)a.R_cap * 4);
  a.a2r = take(A * 4);
  a.Xq = take((size_t)T * d);
  a.tok_sf = take((size_t)T * (d / 32));
  a.Xpq = take((size_t)a.R_cap * d);
  a.xsf = take((size_t)(d / 128) * 32 * Rb * 4);
  a.Hq = take((size_t)a.R_cap * f);
  a.hsf = take((size_t)(f / 128) * 32 * Rb * 4);
  a.Y = take((size_t)a.R_cap * d * 2);
  a.perm_ws = take(permute_ws_bytes(T, k, E_loc));
  a.ffn_ws = take(grouped_ffn_ws_bytes());
  a.total = o;
  return a;
}

}  // namespace vibe

extern "C" const char* vibe_status_string(vibe_status s) {
  switch (s) {
    case VIBE_OK: return "VIBE_OK";
    case VIBE_ERR_INVALID_ARG: return "VIBE_ERR_INVALID_ARG";
    case VIBE_ERR_UNSUPPORTED: return "VIBE_ERR_UNSUPPORTED";
    case VIBE_ERR_WORKSPACE: return "VIBE_ERR_WORKSPACE";
    case VIBE_ERR_CUDA: return "VIBE_ERR_CUDA";
  }
  return "VIBE_ERR_UNKNOWN";
}
extern "C" const char* vibe_last_error(void) { return vibe::g_err; }
extern "C" int32_t vibe_version(void) { return 100; }
extern "C" int64_t vibe_launch_count(void) { return vibe::g_launches; }

extern "C" size_t vibe_workspace_bytes(int32_t which, int32_t T, int32_t k, int32_t E, int32_t E_loc, int32_t d,
                                       int32_t f, int32_t align) {
  using namespace vibe;
  (void)align;
  if (T < 0 || k < 1 || E < 1 || E_loc < 1 || d < 0 || f < 0) return 0;
  switch (which) {
    case VIBE_WS_PERMUTE: return permute_ws_bytes(T, k, E_loc);
    case VIBE_WS_FFN: return grouped_ffn_ws_bytes();
    case VIBE_WS_PROFILE: {
      const size_t R = (size_t)E_loc * (size_t)(T > 0 ? T : 1);
      return round_up(R * d * 2, 256) * 2 + round_up(R * f * 2, 256) + round_up((size_t)(E_loc + 1) * 4, 256) +
             round_up(grouped_ffn_ws_bytes(), 256) + kProfileFlushBytes;
    }
    case VIBE_WS_LAYER: return layer_arena(T, k, E_loc, d, f).total;
    case VIBE_WS_LAYER_FP8: return layer_arena_fp8(T, k, E_loc, d, f).total;
    case VIBE_WS_LAYER_MXFP8: return (d % 128 || f % 128 || d < 128 || f < 128) ? 0 : layer_arena_mx(T, k, E_loc, d, f).total;
    case VIBE_WS_LAYER_HOST:
      return layer_arena(T, k, E_loc, d, f).total + round_up((size_t)T * E * 4, 256) +
             round_up((size_t)T * d * 2, 256) * 2 + round_up((size_t)E * 4, 256) +
             round_up((size_t)8 * E * 4, 256);  // + per-chunk histograms of the pipelined entry
    default: return 0;
  }
}
