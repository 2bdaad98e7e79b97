"""Oracle: the bandit exploration planner of PAPER.md s4.3, stated formula by formula (TEST INFRASTRUCTURE).

  T_plan(a) = d * C * s * t_step ; A = {(d, s) | T_plan <= W}, W = T_train * N_spot
  sigma_all = mean of sigma_g over explored and unexplored groups, sigma_unc = mean over unexplored; r = ratio   (:177-181)
  mu_i = mean of the n_i = min(N_i, W_b) most recent feedbacks of action i                   (:187-189)
  UCB(a_i) = mu_i + beta * sqrt(ln(N + 1) / n_i), N = sum_i N_i ; +inf if n_i = 0            (:193-195)
  a* = argmax UCB; ties -> lower planned cost, fewer steps, fewer sequences                  (:197-199)

Pinned by tests/test_planner.py with values worked out by hand from these formulas.
"""
from __future__ import annotations

import math
from typing import Dict, List, Sequence, Tuple

Action = Tuple[int, int]


def plan_time(a: Action, n_prompts: int, t_step: float) -> float:
    d, s = a
    return d * n_prompts * s * t_step


def eligible(d_values: Sequence[int], s_values: Sequence[int], n_prompts: int, t_step: float, t_train: float,
             n_spot: float) -> List[Action]:
    W = t_train * n_spot
    return [(d, s) for d in d_values for s in s_values if plan_time((d, s), n_prompts, t_step) <= W]


def feedback(sigma_cov: Sequence[float], sigma_unc: Sequence[float]) -> float:
    sigma_all = (sum(sigma_cov) + sum(sigma_unc)) / (len(sigma_cov) + len(sigma_unc))
    sigma_unc_mean = sum(sigma_unc) / len(sigma_unc)
    return sigma_all / sigma_unc_mean


class Planner:
    def __init__(self, d_values, s_values, n_prompts: int, t_step: float, beta: float, window: int):
        self.d_values, self.s_values = list(d_values), list(s_values)
        self.n_prompts, self.t_step, self.beta, self.window = n_prompts, t_step, beta, window
        self.history: Dict[Action, List[float]] = {(d, s): [] for d in self.d_values for s in self.s_values}

    def ucb(self, a: Action) -> float:
        hist = self.history[a]
        n_i = min(len(hist), self.window)
        if n_i == 0:
            return math.inf
        N = sum(len(h) for h in self.history.values())
        mu = sum(hist[-n_i:]) / n_i
        return mu + self.beta * math.sqrt(math.log(N + 1) / n_i)

    def select(self, t_train: float, n_spot: float) -> Tuple[Action, float]:
        cands = eligible(self.d_values, self.s_values, self.n_prompts, self.t_step, t_train, n_spot)
        if not cands:
            raise ValueError("no eligible action")
        best = sorted(cands, key=lambda a: (-self.ucb(a), plan_time(a, self.n_prompts, self.t_step), a[1], a[0]))[0]
        return best, self.ucb(best)

    def update(self, a: Action, r: float) -> None:
        self.history[a].append(float(r))
