/* spot_planner.h - host-side bandit exploration planner of SPOTLIGHT (single-threaded host code, no GPU).
 *
 * PAPER.md s4.3 (lines 153-199):
 *   action a = (d, s): d sequences per prompt, s effective denoising steps                    (s4.3.1, :155-157)
 *   T_plan(a) = d * C * s * t_step;  eligible set A = {(d, s) | T_plan(d, s) <= W}, W = T_train * N_spot   (:161-167)
 *   feedback r = mean(sigma_g over explored and unexplored groups) / mean(sigma_g over unexplored groups)   (:175-183)
 *   per action: sliding window of the W_b most recent feedbacks, n_i = min(N_i, W_b), mean mu_i             (:187-189)
 *   UCB(a_i) = mu_i + beta * sqrt(ln(N + 1) / n_i), N = sum_i N_i; +inf when n_i = 0                        (:193-195)
 *   a* = argmax UCB, ties -> lower planned cost, then fewer steps, then fewer sequences                     (:197-199)
 * The per-prompt sigma_g come from spot_seed_rewards / spot_explore (d_stats[:, 1]).  The paper gives no value for
 * W_b (reading S17: caller-supplied); beta = 0.5 in the paper (:461, :486).
 * All functions return spot_status; pointers are HOST pointers; the planner object is not thread-safe.
 */
#ifndef SPOT_PLANNER_H_
#define SPOT_PLANNER_H_

#include "spot.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spot_planner spot_planner;
typedef struct { int32_t d, s; } spot_action;

/* Action grid = d_values x s_values (all > 0, each list without duplicates); n_prompts = C; t_step > 0 seconds per
 * denoising step per sequence; beta >= 0 (0 = greedy on the window means; the paper sweeps beta in {0, 0.5, 1.0}); window = W_b >= 1. */
spot_status spot_planner_create(const int32_t *d_values, int n_d, const int32_t *s_values, int n_s, int n_prompts,
                                double t_step, double beta, int window, spot_planner **out);
spot_status spot_planner_destroy(spot_planner *p);

/* Eligible actions for the window W = t_train * n_spot, in (d, s) grid order; writes min(count, cap) actions to out
 * (out may be NULL when cap == 0) and the full count to n_out. */
spot_status spot_planner_eligible(const spot_planner *p, double t_train, double n_spot, spot_action *out, int cap,
                                  int *n_out);
/* UCB choice among the eligible actions.  SPOT_ERR_SHAPE when no action is eligible.  *ucb may be +inf. */
spot_status spot_planner_select(const spot_planner *p, double t_train, double n_spot, spot_action *chosen, double *ucb);
/* r = mean(sigma over cov U unc) / mean(sigma over unc); n_unc >= 1 and mean(unc) > 0 required (else SPOT_ERR_SHAPE). */
spot_status spot_planner_feedback(const float *sigma_cov, int n_cov, const float *sigma_unc, int n_unc, double *r);
/* Record feedback r for action a (must be on the grid): N_i += 1, window keeps the W_b most recent values. */
spot_status spot_planner_update(spot_planner *p, spot_action a, double r);
/* Inspect one action: windowed mean (0 when n_i = 0), n_i, N_i and the total N. Any output may be NULL. */
spot_status spot_planner_stats(const spot_planner *p, spot_action a, double *mean, int *n_i, int64_t *N_i, int64_t *N_total);

#ifdef __cplusplus
}
#endif
#endif /* SPOT_PLANNER_H_ */
