"""Bandit planner (PAPER.md s4.3): pins for oracle/planner.py from hand-worked values of the paper's formulas, and
parity of the host C++ planner in libspot.so (include/spot_planner.h) with the oracle.  CPU only."""
import math
import random

import pytest

import paper_2606_19004_b200 as spot
from oracle import planner as orc
from paper_2606_19004_b200 import build as spot_build


@pytest.fixture(scope="module", autouse=True)
def _lib():
    spot_build.build()


# ------------------------------------------------------------------ pins for the oracle
def test_oracle_eligibility_boundary():
    # T_plan = d * C * s * t_step <= W = T_train * N_spot.  C = 32, t_step = 0.5 s.
    # (16, 12): 16*32*12*0.5 = 3072 s ; W = 384 s * 8 GPUs = 3072 s -> eligible (<=), (16, 20) = 5120 -> not.
    acts = orc.eligible([16, 32], [12, 20], 32, 0.5, 384.0, 8)
    assert acts == [(16, 12)]
    assert orc.eligible([16, 32], [12, 20], 32, 0.5, 384.0 - 1e-9, 8) == []
    assert orc.eligible([16, 32], [12, 20], 32, 0.5, 1280.0, 8) == [(16, 12), (16, 20), (32, 12), (32, 20)]   # 10240 = 32*32*20*0.5


def test_oracle_feedback_ratio_hand_worked():
    # explored sigmas 0.30, 0.50; unexplored 0.10, 0.30 -> all = 1.2/4 = 0.3, unc = 0.2, r = 1.5
    assert abs(orc.feedback([0.30, 0.50], [0.10, 0.30]) - 1.5) < 1e-12
    assert abs(orc.feedback([], [0.2, 0.4]) - 1.0) < 1e-12        # nothing explored: ratio 1


def test_oracle_ucb_hand_worked_and_window():
    p = orc.Planner([8, 16], [12, 20], 4, 1.0, 0.5, window=2)
    assert p.ucb((8, 12)) == math.inf                               # unobserved
    p.update((8, 12), 1.0)
    p.update((8, 12), 1.4)
    p.update((16, 12), 2.0)
    # N = 3; action (8,12): n = 2, mu = 1.2 -> 1.2 + 0.5 * sqrt(ln 4 / 2) = 1.2 + 0.5 * 0.8325546 = 1.6162773
    assert abs(p.ucb((8, 12)) - 1.6162773) < 1e-6
    # action (16,12): n = 1, mu = 2.0 -> 2.0 + 0.5 * sqrt(ln 4) = 2.0 + 0.5 * 1.1774100 = 2.5887050
    assert abs(p.ucb((16, 12)) - 2.5887050) < 1e-6
    p.update((8, 12), 3.0)                                          # window W_b = 2 keeps (1.4, 3.0): mu = 2.2, N = 4
    assert abs(p.ucb((8, 12)) - (2.2 + 0.5 * math.sqrt(math.log(5) / 2))) < 1e-12


def test_oracle_selection_order_and_ties():
    p = orc.Planner([8, 16], [12, 20], 4, 1.0, 0.5, window=4)
    big = (1e9, 1.0)
    # all unobserved (+inf everywhere): lowest planned cost first -> (8,12) cost 384
    assert p.select(*big)[0] == (8, 12)
    p.update((8, 12), 1.0)
    # remaining +inf: (8,20) cost 640, (16,12) cost 768, (16,20) cost 1280 -> (8,20)
    assert p.select(*big)[0] == (8, 20)
    p.update((8, 20), 1.0)
    p.update((16, 12), 1.0)
    assert p.select(*big)[0] == (16, 20)
    p.update((16, 20), 1.0)
    # now every action has n = 1, mu = 1: equal UCB -> ties by cost -> (8,12)
    a, u = p.select(*big)
    assert a == (8, 12) and abs(u - (1.0 + 0.5 * math.sqrt(math.log(5)))) < 1e-12
    # equal cost, different shape: C*t_step = 1 -> (2,6) and (3,4) and (4,3) all cost 12: fewer steps first -> (4,3)
    q = orc.Planner([2, 3, 4], [3, 4, 6], 1, 1.0, 0.5, window=4)
    for a in q.history:
        q.update(a, 1.0)
    cands = [a for a in q.history if orc.plan_time(a, 1, 1.0) == 12]
    assert sorted(cands) == [(2, 6), (3, 4), (4, 3)]
    assert q.select(12.0, 1.0)[0] in q.history
    only12 = orc.Planner([2, 3, 4], [3, 4, 6], 1, 1.0, 0.5, window=4)
    for a in only12.history:
        if orc.plan_time(a, 1, 1.0) != 12:
            only12.update(a, -100.0)        # make every other action unattractive
        else:
            only12.update(a, 1.0)
    assert only12.select(1e9, 1.0)[0] == (4, 3)
    # restricted budget: with W = 400 only (8,12) is eligible
    assert p.select(100.0, 4.0)[0] == (8, 12)
    with pytest.raises(ValueError):
        p.select(1.0, 1.0)


# ------------------------------------------------------------------ C++ planner vs oracle
def test_c_planner_matches_oracle_on_random_run():
    rng = random.Random(2606)
    d_vals, s_vals = [4, 8, 16, 32], [12, 14, 16, 20]
    cp = spot.Planner(d_vals, s_vals, 28, 0.37, beta=0.5, window=3)
    op = orc.Planner(d_vals, s_vals, 28, 0.37, 0.5, 3)
    for it in range(300):
        t_train, n_spot = rng.uniform(100, 2500), rng.choice([1, 2, 4, 8])
        want = orc.eligible(d_vals, s_vals, 28, 0.37, t_train, n_spot)
        assert cp.spot_planner_eligible(t_train, n_spot) == want
        if not want:
            with pytest.raises(spot.SpotError):
                cp.spot_planner_select(t_train, n_spot)
            continue
        a_c, u_c = cp.spot_planner_select(t_train, n_spot)
        a_o, u_o = op.select(t_train, n_spot)
        assert a_c == a_o, it
        assert (math.isinf(u_c) and math.isinf(u_o)) or abs(u_c - u_o) < 1e-12
        sig_cov = [rng.uniform(0.05, 1.0) for _ in range(28)]
        sig_unc = [rng.uniform(0.05, 0.6) for _ in range(4)]          # 4 unexplored prompts per iteration
        r_c = spot.spot_planner_feedback(sig_cov, sig_unc)
        import numpy as np
        r_o = orc.feedback([float(np.float32(x)) for x in sig_cov], [float(np.float32(x)) for x in sig_unc])
        assert abs(r_c - r_o) < 1e-12
        cp.spot_planner_update(a_c, r_c)
        op.update(a_o, r_o)
        st = cp.spot_planner_stats(a_c)
        assert st["N"] == sum(len(h) for h in op.history.values())
        assert st["n_i"] == min(len(op.history[a_o]), 3)
        assert abs(st["mean"] - sum(op.history[a_o][-3:]) / st["n_i"]) < 1e-12


def test_beta_zero_is_greedy_on_window_means():
    """PAPER.md:486 sweeps beta in {0, 0.5, 1.0}: beta = 0 is accepted and selects the best window mean (after every
    action was tried once: untried actions still score +inf)."""
    d_vals, s_vals = [4, 8], [12, 16]
    cp = spot.Planner(d_vals, s_vals, 8, 1.0, beta=0.0, window=2)
    op = orc.Planner(d_vals, s_vals, 8, 1.0, 0.0, 2)
    fb = {(4, 12): 1.0, (8, 12): 1.4, (4, 16): 1.2, (8, 16): 1.3}
    for it in range(8):
        a_c, u_c = cp.spot_planner_select(1e6, 8)
        a_o, u_o = op.select(1e6, 8)
        assert a_c == a_o
        if it >= 4:
            assert a_c == (8, 12) and abs(u_c - 1.4) < 1e-12 and abs(u_o - 1.4) < 1e-12      # no exploration bonus
        cp.spot_planner_update(a_c, fb[a_c])
        op.update(a_o, fb[a_o])
    with pytest.raises(spot.SpotError):
        spot.Planner(d_vals, s_vals, 8, 1.0, beta=-0.1)
    with pytest.raises(spot.SpotError):
        spot.Planner(d_vals, s_vals, 8, 1.0, beta=float("nan"))


def test_c_planner_argument_errors():
    with pytest.raises(spot.SpotError):
        spot.Planner([4, 4], [12], 8, 1.0)                 # duplicate d
    with pytest.raises(spot.SpotError):
        spot.Planner([4], [12], 8, 0.0)                    # t_step must be > 0
    p = spot.Planner([4], [12], 8, 1.0)
    with pytest.raises(spot.SpotError):
        p.spot_planner_update((5, 12), 1.0)                # not on the grid
    with pytest.raises(spot.SpotError):
        spot.spot_planner_feedback([0.1], [])              # needs unexplored groups
