// Adaptive redundancy allocation (§4.2.2, App. B Eq. 6-9, App. C Alg. 1): the step
// immediately upstream of the rollout.  Host code: a batch is N <= a few hundred prompts and the plan feeds darts_prefill's
// host-side Kp array, so there is nothing for the GPU to do.  Written from the paper; shares nothing with oracle/allocation.py.
#include <math.h>

#include <vector>

#include "darts.h"

extern "C" {

// sigma~^2 <- (1 - beta) sigma~^2 + beta sigma^2 (EMA); entries < 0 mean "no history yet".
darts_status darts_update_variance_ema(float *var_ema_host, const float *len_var_host, int32_t G, float beta) {
  if (!var_ema_host || !len_var_host || G <= 0 || !(beta >= 0.f && beta <= 1.f)) return DARTS_ERR_INVALID_ARG;
  for (int i = 0; i < G; ++i) {
    double old = var_ema_host[i], obs = len_var_host[i];
    var_ema_host[i] = (float)(old < 0 ? obs : (1.0 - (double)beta) * old + (double)beta * obs);
  }
  return DARTS_OK;
}

// Eq. 8-9: M* = rho / (lambda k);  M_total = clip(floor(M*), K G, 2 K G).
darts_status darts_redundancy_budget(double rho, double lambda, double k, int32_t G, int32_t K, int64_t *M_total_out) {
  if (!M_total_out || G <= 0 || K <= 0 || !(lambda > 0) || !(k > 0) || !(rho >= 0)) return DARTS_ERR_INVALID_ARG;
  double m = floor(rho / (lambda * k));
  int64_t lo = (int64_t)K * G, hi = 2 * lo;
  *M_total_out = m < (double)lo ? lo : (m > (double)hi ? hi : (int64_t)m);
  return DARTS_OK;
}

// Alg. 1: weights = min-max normalised sigma~_L over the batch (all equal -> 1), greedy on the marginal gain
// w_i (1/M'_i - 1/(M'_i + 1)) among prompts below M_up, ties -> smallest i.  Kp_out sums to min(M_total, G * M_up).
darts_status darts_allocate_redundancy(const float *var_ema_host, int32_t G, int64_t M_total, int32_t M_low, int32_t M_up, int32_t *Kp_out_host) {
  if (!var_ema_host || !Kp_out_host || G <= 0 || M_low <= 0 || M_up < M_low || M_total < (int64_t)G * M_low) return DARTS_ERR_INVALID_ARG;
  std::vector<double> w(G);
  double lo = INFINITY, hi = -INFINITY;
  for (int i = 0; i < G; ++i) {
    if (!(var_ema_host[i] >= 0.f)) return DARTS_ERR_INVALID_ARG;
    w[i] = sqrt((double)var_ema_host[i]);
    lo = fmin(lo, w[i]); hi = fmax(hi, w[i]);
  }
  for (int i = 0; i < G; ++i) w[i] = hi == lo ? 1.0 : (w[i] - lo) / (hi - lo);
  for (int i = 0; i < G; ++i) Kp_out_host[i] = M_low;
  for (int64_t remain = M_total - (int64_t)G * M_low; remain > 0; --remain) {
    double best = -1.0;
    int k = -1;
    for (int i = 0; i < G; ++i)
      if (Kp_out_host[i] < M_up) {
        double m = Kp_out_host[i], gain = w[i] * (1.0 / m - 1.0 / (m + 1.0));
        if (gain > best) { best = gain; k = i; }
      }
    if (k < 0) break;
    Kp_out_host[k] += 1;
  }
  return DARTS_OK;
}

}  // extern "C"
