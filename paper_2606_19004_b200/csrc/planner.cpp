// planner.cpp - host bandit planner (include/spot_planner.h; PAPER.md s4.3).  Plain C++, no CUDA.
#include <math.h>

#include <deque>
#include <limits>
#include <new>
#include <vector>

#include "../../include/spot_planner.h"

struct spot_planner {
  std::vector<int32_t> d_vals, s_vals;
  int n_prompts;
  double t_step, beta;
  int window;
  std::vector<std::deque<double>> recent;   // per action, the W_b most recent feedbacks (oldest first)
  std::vector<int64_t> count;               // N_i
  int64_t total;                            // N
  int index(spot_action a) const {
    for (size_t i = 0; i < d_vals.size(); ++i)
      for (size_t j = 0; j < s_vals.size(); ++j)
        if (d_vals[i] == a.d && s_vals[j] == a.s) return (int)(i * s_vals.size() + j);
    return -1;
  }
  double plan_time(int32_t d, int32_t s) const { return (double)d * (double)n_prompts * (double)s * t_step; }
};

extern "C" {

spot_status spot_planner_create(const int32_t* d_values, int n_d, const int32_t* s_values, int n_s, int n_prompts,
                                double t_step, double beta, int window, spot_planner** out) {
  if (!d_values || !s_values || !out) return SPOT_ERR_NULL;
  *out = nullptr;
  if (n_d <= 0 || n_s <= 0 || n_prompts <= 0 || !(t_step > 0.0) || !(beta >= 0.0) || window < 1) return SPOT_ERR_SHAPE;
  for (int i = 0; i < n_d; ++i) {
    if (d_values[i] <= 0) return SPOT_ERR_SHAPE;
    for (int j = 0; j < i; ++j) if (d_values[j] == d_values[i]) return SPOT_ERR_SHAPE;
  }
  for (int i = 0; i < n_s; ++i) {
    if (s_values[i] <= 0) return SPOT_ERR_SHAPE;
    for (int j = 0; j < i; ++j) if (s_values[j] == s_values[i]) return SPOT_ERR_SHAPE;
  }
  spot_planner* p = new (std::nothrow) spot_planner();
  if (!p) return SPOT_ERR_CUDA;
  p->d_vals.assign(d_values, d_values + n_d);
  p->s_vals.assign(s_values, s_values + n_s);
  p->n_prompts = n_prompts; p->t_step = t_step; p->beta = beta; p->window = window;
  p->recent.resize((size_t)n_d * n_s);
  p->count.assign((size_t)n_d * n_s, 0);
  p->total = 0;
  *out = p;
  return SPOT_OK;
}

spot_status spot_planner_destroy(spot_planner* p) {
  if (!p) return SPOT_ERR_NULL;
  delete p;
  return SPOT_OK;
}

spot_status spot_planner_eligible(const spot_planner* p, double t_train, double n_spot, spot_action* out, int cap,
                                  int* n_out) {
  if (!p || !n_out || (cap > 0 && !out)) return SPOT_ERR_NULL;
  if (cap < 0 || !(t_train >= 0.0) || !(n_spot >= 0.0)) return SPOT_ERR_SHAPE;
  const double W = t_train * n_spot;
  int n = 0;
  for (int32_t d : p->d_vals)
    for (int32_t s : p->s_vals)
      if (p->plan_time(d, s) <= W) {
        if (n < cap) { out[n].d = d; out[n].s = s; }
        ++n;
      }
  *n_out = n;
  return SPOT_OK;
}

spot_status spot_planner_select(const spot_planner* p, double t_train, double n_spot, spot_action* chosen, double* ucb) {
  if (!p || !chosen) return SPOT_ERR_NULL;
  if (!(t_train >= 0.0) || !(n_spot >= 0.0)) return SPOT_ERR_SHAPE;
  const double W = t_train * n_spot;
  bool have = false;
  double best_u = 0.0, best_cost = 0.0;
  spot_action best{0, 0};
  for (size_t i = 0; i < p->d_vals.size(); ++i)
    for (size_t j = 0; j < p->s_vals.size(); ++j) {
      const int32_t d = p->d_vals[i], s = p->s_vals[j];
      const double cost = p->plan_time(d, s);
      if (!(cost <= W)) continue;
      const std::deque<double>& win = p->recent[i * p->s_vals.size() + j];
      double u;
      if (win.empty()) {
        u = std::numeric_limits<double>::infinity();
      } else {
        double sum = 0.0;
        for (double r : win) sum += r;
        u = sum / (double)win.size() + p->beta * sqrt(log((double)p->total + 1.0) / (double)win.size());
      }
      bool better = !have || u > best_u;
      if (have && u == best_u) {             // ties: lower planned cost, then fewer steps, then fewer sequences
        if (cost != best_cost) better = cost < best_cost;
        else if (s != best.s) better = s < best.s;
        else better = d < best.d;
      }
      if (better) { have = true; best_u = u; best_cost = cost; best.d = d; best.s = s; }
    }
  if (!have) return SPOT_ERR_SHAPE;
  *chosen = best;
  if (ucb) *ucb = best_u;
  return SPOT_OK;
}

spot_status spot_planner_feedback(const float* sigma_cov, int n_cov, const float* sigma_unc, int n_unc, double* r) {
  if (!r || !sigma_unc || (n_cov > 0 && !sigma_cov)) return SPOT_ERR_NULL;
  if (n_cov < 0 || n_unc < 1) return SPOT_ERR_SHAPE;
  double all = 0.0, unc = 0.0;
  for (int i = 0; i < n_cov; ++i) all += (double)sigma_cov[i];
  for (int i = 0; i < n_unc; ++i) unc += (double)sigma_unc[i];
  all = (all + unc) / (double)(n_cov + n_unc);
  unc /= (double)n_unc;
  if (!(unc > 0.0)) return SPOT_ERR_SHAPE;
  *r = all / unc;
  return SPOT_OK;
}

spot_status spot_planner_update(spot_planner* p, spot_action a, double r) {
  if (!p) return SPOT_ERR_NULL;
  const int i = p->index(a);
  if (i < 0 || !(r == r)) return SPOT_ERR_SHAPE;
  std::deque<double>& win = p->recent[i];
  win.push_back(r);
  while ((int)win.size() > p->window) win.pop_front();
  ++p->count[i];
  ++p->total;
  return SPOT_OK;
}

spot_status spot_planner_stats(const spot_planner* p, spot_action a, double* mean, int* n_i, int64_t* N_i, int64_t* N_total) {
  if (!p) return SPOT_ERR_NULL;
  const int i = p->index(a);
  if (i < 0) return SPOT_ERR_SHAPE;
  const std::deque<double>& win = p->recent[i];
  double sum = 0.0;
  for (double r : win) sum += r;
  if (mean) *mean = win.empty() ? 0.0 : sum / (double)win.size();
  if (n_i) *n_i = (int)win.size();
  if (N_i) *N_i = p->count[i];
  if (N_total) *N_total = p->total;
  return SPOT_OK;
}

}  // extern "C"
