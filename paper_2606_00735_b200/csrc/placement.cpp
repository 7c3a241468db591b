// placement.cpp -- host-side placement evaluator and greedy solvers (a7, a8), fp64.
//   T = max_g f_g(n_g),  n_g = sum_{e in S_g} w_e
//   s_g = 1/f_g(n_ref), tau_g = N s_g / sum_h s_h, descending-load assignment to the GPU
//   farthest below its target                                   (L186-L196; Alg. 1)
// with f_g(n) = f(n)/sigma_g (M5) and f from the measured profile (M1).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>

#include <algorithm>
#include <numeric>
#include <vector>

#include "../../include/vibe.h"

namespace vibe {
void set_error(const char* fmt, ...);
void clear_error();

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
