// placement.cpp -- host-side placement evaluator and greedy solvers (a7, a8), fp64.
//   T = max_g f_g(n_g),  n_g = sum_{e in S_g} w_e
//   s_g = 1/f_g(n_ref), tau_g = N s_g / sum_h s_h, descending-load assignment to the GPU
//   farthest below its target                                   (L186-L196; Alg. 1)
// with f_g(n) = f(n)/sigma_g (M5) and f from the measured profile (M1).
// f1: drift detector  d = 1 - w.w_ref/(|w||w_ref|)  (L202-L208; Alg. 1 phase 3, L454-L462)
// and the incremental swap solver (Algorithm 2; prose L210-L214, L426-L428).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>

#include <algorithm>
#include <deque>
#include <new>
#include <numeric>
#include <vector>

#include "../../include/vibe.h"

namespace vibe {
void set_error(const char* fmt, ...);
void clear_error();
}
#define VIBE_REQUIRE_HOST(cond, ...)      \
  do {                                    \
    if (!(cond)) {                        \
      ::vibe::set_error(__VA_ARGS__);     \
      return VIBE_ERR_INVALID_ARG;        \
    }                                     \
  } while (0)
namespace vibe {

namespace {
struct Model {
  std::vector<double> t, l;  // with the origin prepended, running max applied
  int E_prof = 1;
  bool linear = false;       // NULL model: f(n) = n

  bool init(const vibe_latency_model* m) {
    if (m == nullptr) {
      linear = true;
      return true;
    }
    if (m->n_points < 1 || !m->tokens || !m->latency_us || m->E_prof < 1) return false;
    t.assign(1, 0.0);
    l.assign(1, 0.0);
    double run = 0.0;
    for (int i = 0; i < m->n_points; ++i) {
      if (!(m->tokens[i] > t.back())) return false;
      run = std::max(run, m->latency_us[i]);
      t.push_back(m->tokens[i]);
      l.push_back(run);
    }
    E_prof = m->E_prof;
    return true;
  }
  double per_expert(double n) const {
    if (linear) return n > 0 ? n : 0.0;
    if (n <= 0.0) return 0.0;
    const size_t last = t.size() - 1;
    if (n >= t[last]) {
      const double slope = (l[last] - l[last - 1]) / (t[last] - t[last - 1]);
      return l[last] + slope * (n - t[last]);
    }
    size_t i = (size_t)(std::upper_bound(t.begin(), t.end(), n) - t.begin()) - 1;
    return l[i] + (l[i + 1] - l[i]) * (n - t[i]) / (t[i + 1] - t[i]);
  }
  double whole_kernel(double n_total) const {
    if (linear) return n_total > 0 ? n_total : 0.0;
    return E_prof * per_expert(n_total / E_prof);
  }
};

vibe_status greedy(const double* load, int E, int G, const double* scale, const Model& m, int cap, int32_t* assign) {
  double N = 0.0;
  for (int e = 0; e < E; ++e) N += load[e];
  const double fref = m.whole_kernel(N / E);
  std::vector<double> s(G), tau(G), n(G, 0.0);
  std::vector<int> cnt(G, 0);
  double ssum = 0.0;
  for (int g = 0; g < G; ++g) {
    const double sg = scale ? scale[g] : 1.0;
    s[g] = fref > 0.0 ? 1.0 / (fref / sg) : sg;
    ssum += s[g];
  }
  for (int g = 0; g < G; ++g) tau[g] = N * s[g] / ssum;
  std::vector<int> order(E);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return load[a] > load[b]; });
  for (int e : order) {
    int best = -1;
    double best_gap = 0.0;
    for (int g = 0; g < G; ++g) {
      if (cap > 0 && cnt[g] >= cap) continue;
      const double gap = tau[g] - n[g];
      if (best < 0 || gap > best_gap) {
        best = g;
        best_gap = gap;
      }
    }
    if (best < 0) {
      set_error("vibe_placement_greedy: cap*G < E");
      return VIBE_ERR_INVALID_ARG;
    }
    assign[e] = best;
    n[best] += load[e];
    cnt[best] += 1;
  }
  return VIBE_OK;
}
}  // namespace
}  // namespace vibe

extern "C" double vibe_placement_eval(const int32_t* assign, const double* load, int32_t E, int32_t G,
                                      const double* scale, const vibe_latency_model* m, int32_t model_kind,
                                      double* per_bin) {
  using namespace vibe;
  clear_error();
  if (!assign || !load || !scale || E < 1 || G < 1 || (model_kind != VIBE_MODEL_A && model_kind != VIBE_MODEL_B)) {
    set_error("vibe_placement_eval: invalid arguments");
    return -1.0;
  }
  Model mod;
  if (!mod.init(m)) {
    set_error("vibe_placement_eval: invalid latency model");
    return -1.0;
  }
  std::vector<double> acc(G, 0.0);
  for (int e = 0; e < E; ++e) {
    const int g = assign[e];
    if (g < 0 || g >= G) {
      set_error("vibe_placement_eval: assign[%d] = %d out of range", e, g);
      return -1.0;
    }
    acc[g] += (model_kind == VIBE_MODEL_A) ? load[e] : mod.per_expert(load[e]);
  }
  double worst = 0.0;
  for (int g = 0; g < G; ++g) {
    if (!(scale[g] > 0.0)) {
      set_error("vibe_placement_eval: scale[%d] <= 0", g);
      return -1.0;
    }
    const double L = (model_kind == VIBE_MODEL_A) ? mod.whole_kernel(acc[g]) : acc[g];
    const double v = L / scale[g];
    if (per_bin) per_bin[g] = v;
    worst = std::max(worst, v);
  }
  return worst;
}

extern "C" vibe_status vibe_placement_greedy(const double* load, int32_t E, int32_t G, const double* scale,
                                             const vibe_latency_model* m, int32_t cap, int32_t* assign) {
  using namespace vibe;
  clear_error();
  if (!load || !scale || !assign || E < 1 || G < 1 || cap < 0) {
    set_error("vibe_placement_greedy: invalid arguments");
    return VIBE_ERR_INVALID_ARG;
  }
  for (int g = 0; g < G; ++g)
    if (!(scale[g] > 0.0)) {
      set_error("vibe_placement_greedy: scale[%d] <= 0", g);
      return VIBE_ERR_INVALID_ARG;
    }
  Model mod;
  if (!mod.init(m)) {
    set_error("vibe_placement_greedy: invalid latency model");
    return VIBE_ERR_INVALID_ARG;
  }
  return greedy(load, E, G, scale, mod, cap, assign);
}

extern "C" vibe_status vibe_placement_token_balanced(const double* load, int32_t E, int32_t G, int32_t cap,
                                                     int32_t* assign) {
  using namespace vibe;
  clear_error();
  if (!load || !assign || E < 1 || G < 1 || cap < 0) {
    set_error("vibe_placement_token_balanced: invalid arguments");
    return VIBE_ERR_INVALID_ARG;
  }
  Model mod;
  mod.init(nullptr);
  return greedy(load, E, G, nullptr, mod, cap, assign);
}

extern "C" vibe_status vibe_placement_contiguous(int32_t E, int32_t G, int32_t* assign) {
  using namespace vibe;
  clear_error();
  if (!assign || E < 1 || G < 1) {
    set_error("vibe_placement_contiguous: invalid arguments");
    return VIBE_ERR_INVALID_ARG;
  }
  for (int e = 0; e < E; ++e) assign[e] = (int32_t)(((int64_t)e * G) / E);
  return VIBE_OK;
}

// ======================================================================================
// f1: drift detection and incremental update
// ======================================================================================
namespace vibe {
namespace {
double cosine_distance(const double* w, const double* r, int E) {
  double dot = 0.0, nw = 0.0, nr = 0.0;
  for (int e = 0; e < E; ++e) {
    dot += w[e] * r[e];
    nw += w[e] * w[e];
    nr += r[e] * r[e];
  }
  if (nw == 0.0 || nr == 0.0) return 0.0;  // D1: a zero vector carries no direction
  return 1.0 - dot / (sqrt(nw) * sqrt(nr));
}

// latency of one bin, members summed in ascending expert index
double bin_latency(const int32_t* assign, const double* load, const std::vector<double>& per, int E, int g,
                   double sigma, const Model& m, int kind) {
  double acc = 0.0;
  for (int e = 0; e < E; ++e)
    if (assign[e] == g) acc += (kind == VIBE_MODEL_A) ? load[e] : per[e];
  return ((kind == VIBE_MODEL_A) ? m.whole_kernel(acc) : acc) / sigma;
}
}  // namespace
}  // namespace vibe

struct vibe_drift_monitor {
  int L, E, window, H;
  double delta;
  std::deque<std::vector<double>> samples;  // oldest first, each L*E
  std::vector<double> ref;
  bool has_ref = false;
  long long passes = 0;
  int cooldown = 0;
  void mean(double* W) const {
    const size_t n = (size_t)L * E;
    for (size_t i = 0; i < n; ++i) W[i] = 0.0;
    for (const auto& s : samples)
      for (size_t i = 0; i < n; ++i) W[i] += s[i];
    const double cnt = samples.empty() ? 1.0 : (double)samples.size();
    for (size_t i = 0; i < n; ++i) W[i] /= cnt;
  }
};

extern "C" double vibe_drift_cosine(const double* w, const double* w_ref, int32_t E) {
  using namespace vibe;
  clear_error();
  if (!w || !w_ref || E < 1) {
    set_error("vibe_drift_cosine: invalid arguments");
    return -1.0;
  }
  return cosine_distance(w, w_ref, E);
}

extern "C" vibe_drift_monitor* vibe_drift_monitor_create(int32_t L, int32_t E, int32_t window, int32_t H,
                                                         double delta) {
  using namespace vibe;
  clear_error();
  if (L < 1 || E < 1 || window < 1 || H < 1 || !(delta >= 0.0)) {
    set_error("vibe_drift_monitor_create: need L, E, window, H >= 1 and delta >= 0");
    return nullptr;
  }
  vibe_drift_monitor* m = new (std::nothrow) vibe_drift_monitor();
  if (!m) {
    set_error("vibe_drift_monitor_create: out of memory");
    return nullptr;
  }
  m->L = L;
  m->E = E;
  m->window = window;
  m->H = H;
  m->delta = delta;
  return m;
}

extern "C" void vibe_drift_monitor_destroy(vibe_drift_monitor* m) { delete m; }

extern "C" vibe_status vibe_drift_monitor_set_reference(vibe_drift_monitor* m, const double* W) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE_HOST(m && W, "vibe_drift_monitor_set_reference: NULL argument");
  m->ref.assign(W, W + (size_t)m->L * m->E);
  m->has_ref = true;
  return VIBE_OK;
}

extern "C" vibe_status vibe_drift_monitor_rearranged(vibe_drift_monitor* m) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE_HOST(m, "vibe_drift_monitor_rearranged: NULL monitor");
  m->ref.resize((size_t)m->L * m->E);
  m->mean(m->ref.data());
  m->has_ref = true;
  m->cooldown = m->H;
  return VIBE_OK;
}

extern "C" vibe_status vibe_drift_monitor_window_mean(const vibe_drift_monitor* m, double* W) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE_HOST(m && W, "vibe_drift_monitor_window_mean: NULL argument");
  m->mean(W);
  return VIBE_OK;
}

extern "C" int32_t vibe_drift_monitor_push(vibe_drift_monitor* m, const double* loads, double* d_out,
                                           int32_t* checked) {
  using namespace vibe;
  clear_error();
  if (checked) *checked = 0;
  if (!m || !loads) {
    set_error("vibe_drift_monitor_push: NULL argument");
    return -1;
  }
  const size_t n = (size_t)m->L * m->E;
  m->samples.emplace_back(loads, loads + n);
  if ((int)m->samples.size() > m->window) m->samples.pop_front();
  m->passes += 1;
  if (m->cooldown > 0) {
    m->cooldown -= 1;
    return 0;
  }
  if (!m->has_ref || m->passes % m->H != 0) return 0;
  std::vector<double> w(n);
  m->mean(w.data());
  double worst = 0.0;
  for (int l = 0; l < m->L; ++l) {
    const double d = cosine_distance(w.data() + (size_t)l * m->E, m->ref.data() + (size_t)l * m->E, m->E);
    if (d_out) d_out[l] = d;
    if (l == 0 || d > worst) worst = d;
  }
  if (checked) *checked = 1;
  return worst > m->delta ? 1 : 0;
}

extern "C" vibe_status vibe_placement_swap_refine(int32_t* assign, const double* load, int32_t E, int32_t G,
                                                  const double* scale, const vibe_latency_model* m,
                                                  int32_t model_kind, double eps, int32_t max_swaps,
                                                  int32_t* n_swaps, int32_t* swaps) {
  using namespace vibe;
  clear_error();
  if (n_swaps) *n_swaps = 0;
  VIBE_REQUIRE_HOST(assign && load && scale && E >= 1 && G >= 1 && max_swaps >= 0 && eps >= 0.0 &&
                        (model_kind == VIBE_MODEL_A || model_kind == VIBE_MODEL_B),
                    "vibe_placement_swap_refine: invalid arguments");
  for (int e = 0; e < E; ++e)
    VIBE_REQUIRE_HOST(assign[e] >= 0 && assign[e] < G, "vibe_placement_swap_refine: assign[%d] out of range", e);
  for (int g = 0; g < G; ++g) VIBE_REQUIRE_HOST(scale[g] > 0.0, "vibe_placement_swap_refine: scale[%d] <= 0", g);
  Model mod;
  VIBE_REQUIRE_HOST(mod.init(m), "vibe_placement_swap_refine: invalid latency model");
  std::vector<double> per(E), Lg(G);
  for (int e = 0; e < E; ++e) per[e] = mod.per_expert(load[e]);
  int done = 0;
  while (done < max_swaps) {
    double mean = 0.0;
    for (int g = 0; g < G; ++g) {
      Lg[g] = bin_latency(assign, load, per, E, g, scale[g], mod, model_kind);
      mean += Lg[g];
    }
    mean /= G;
    int hi = 0, lo = 0;
    for (int g = 1; g < G; ++g) {
      if (Lg[g] > Lg[hi]) hi = g;   // first maximum / first minimum: ties -> lower g
      if (Lg[g] < Lg[lo]) lo = g;
    }
    if (Lg[hi] <= (1.0 + eps) * mean || hi == lo) break;
    const double before = std::max(Lg[hi], Lg[lo]);
    int bi = -1, bj = -1;
    double best = 0.0;
    for (int ei = 0; ei < E; ++ei) {
      if (assign[ei] != hi) continue;
      for (int ej = 0; ej < E; ++ej) {
        if (assign[ej] != lo) continue;
        assign[ei] = lo;
        assign[ej] = hi;
        const double a = bin_latency(assign, load, per, E, hi, scale[hi], mod, model_kind);
        const double b = bin_latency(assign, load, per, E, lo, scale[lo], mod, model_kind);
        assign[ei] = hi;
        assign[ej] = lo;
        const double red = before - std::max(a, b);
        if (red > best) {          // strict: ties -> lowest (e_i, e_j)
          best = red;
          bi = ei;
          bj = ej;
        }
      }
    }
    if (bi < 0) break;             // "no latency reduction"
    assign[bi] = lo;
    assign[bj] = hi;
    if (swaps) {
      swaps[2 * done] = bi;
      swaps[2 * done + 1] = bj;
    }
    ++done;
  }
  if (n_swaps) *n_swaps = done;
  return VIBE_OK;
}
