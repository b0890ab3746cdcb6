"""Pins of the serving-simulation oracle (oracle/laser_sim_oracle.c; SURVEY §8 f NEXT-4) against what
queueing theory and the paper fix - closed forms, hand-computed values, a library routine and
invariants; none re-types the oracle's loop.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from paper_2606_31580_b200 import workloads as wl


def _fifo_closed_form(arrival, service):
    """Departure times of a single-server FIFO queue WITHOUT a recursion: f_i = max over j <= i of
    (a_j + S_j + ... + S_i) - the busy period that contains i started at some arrival j."""
    cs = np.concatenate([[0.0], np.cumsum(service)])
    # a_j + (cs[i+1] - cs[j])  ->  cs[i+1] + max_j (a_j - cs[j])
    return cs[1:] + np.maximum.accumulate(arrival - cs[:-1])


def _pool_const(S=1, K=4, chunk=0.5, conf=0.5, prompt=100, pre=0.1, conc=0.2):
    return dict(chunk_time=np.full((S, K), chunk, np.float32), conf=np.full((S, K), conf, np.float32),
                prompt_tokens=np.full(S, prompt, np.int32), t_prefill=np.full(S, pre, np.float32),
                t_conclusion=np.full(S, conc, np.float32))


def test_S1_certain_answers_exit_after_one_chunk_and_queue_is_fifo():
    """conf = 1 everywhere exceeds every admissible threshold (lambda_max = 0.97): each request
    generates exactly one chunk, so its service time is known and the finish times must equal the
    closed form of a FIFO single-server queue."""
    pool = wl.sim_pool(S=200, K=15, seed=5)
    pool["conf"][:] = 1.0
    arr = wl.sim_arrivals_poisson(1, 3000, 1.2, seed=6)[:, 0]
    sid = wl.sim_sample_ids(1, 3000, 200, seed=7)[:, 0]
    r = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy())
    assert np.all(r["chunks"] == 1) and np.all(r["exited"] == 1)
    svc = (pool["t_prefill"][sid].astype(np.float64) + pool["chunk_time"][sid, 0].astype(np.float64)
           + pool["t_conclusion"][sid].astype(np.float64))
    np.testing.assert_allclose(r["finish"], _fifo_closed_form(arr, svc), rtol=0, atol=1e-8)
    assert np.all(np.diff(r["finish"]) > 0) and np.all(r["finish"] > arr)


@pytest.mark.parametrize("K_fixed", [1, 7, 15, 40])
def test_S2_vanilla_generates_the_whole_budget(K_fixed):
    """early_exit = 0 (Vanilla): every request generates min(fixed budget, K) chunks."""
    pool = wl.sim_pool(S=50, K=15, seed=8)
    arr = wl.sim_arrivals_poisson(1, 500, 0.2, seed=9)[:, 0]
    sid = wl.sim_sample_ids(1, 500, 50, seed=10)[:, 0]
    r = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy(early_exit=0, adaptive_budget=0, fixed_budget=K_fixed))
    k = min(K_fixed, 15)
    assert np.all(r["chunks"] == k) and np.all(r["exited"] == 0) and np.all(r["budget"] == k)
    svc = (pool["t_prefill"][sid].astype(np.float64) + pool["chunk_time"][sid, :k].astype(np.float64).sum(1)
           + pool["t_conclusion"][sid].astype(np.float64))
    np.testing.assert_allclose(r["finish"], _fifo_closed_form(arr, svc), rtol=0, atol=1e-7)


def test_S3_md1_mean_wait_is_pollaczek_khinchine():
    """Poisson arrivals, deterministic service s (one sample, one chunk): the mean waiting time of
    M/D/1 is rho * s / (2 (1 - rho))."""
    s = 0.1 + 0.5 + 0.2
    rho = 0.7
    n = 400_000
    arr = wl.sim_arrivals_poisson(1, n, rho / s, seed=11)[:, 0]
    pool = _pool_const(K=1)
    r = oracle.sim_queue(arr, np.zeros(n, np.int32), pool, oracle.SimPolicy(early_exit=0, adaptive_budget=0, fixed_budget=1))
    svc = float(np.float32(0.1)) + float(np.float32(0.5)) + float(np.float32(0.2))
    wait = (r["finish"] - arr - svc).mean()
    assert abs(wait - rho * s / (2 * (1 - rho))) < 0.03 * rho * s / (2 * (1 - rho))


def test_S4_fixed_threshold_baselines():
    """beta = 0 and no budget allocator = the Fixed-High / Fixed-Low baselines:
    a request stops at its first ATP whose confidence exceeds the constant threshold."""
    pool = wl.sim_pool(S=300, K=15, seed=12)
    arr = wl.sim_arrivals_poisson(1, 2000, 3.0, seed=13)[:, 0]
    sid = wl.sim_sample_ids(1, 2000, 300, seed=14)[:, 0]
    for lam in (0.95, 0.90):
        r = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy(beta=0.0, lambda_base=lam, adaptive_budget=0, fixed_budget=10))
        c = pool["conf"][sid, :10].astype(np.float64)
        hit = c > lam
        first = np.where(hit.any(1), hit.argmax(1) + 1, 10)
        assert np.array_equal(r["chunks"], first)
        assert np.array_equal(r["exited"], hit.any(1).astype(np.uint8))


def test_S5_budget_values_worked_by_hand():
    """Eq. 6-8 with the paper's defaults, worked by hand.
    Alone in the system (L = 1, f_load = 1): |p| = 50 -> f_diff 0.6 -> B = 6; 275 -> 1.5 -> 15;
    162 -> 0.6 + 112/225 * 0.9 = 1.048 -> floor(10.48) = 10.
    Thirty requests arriving together (request i starts with L = 30 - i in the system), |p| = 162:
    L = 30 -> f_load 1/3 -> floor(3.49) = 3; L = 20 -> floor(5.24) = 5; L = 15 -> floor(6.98) = 6;
    L <= 10 -> 10.  |p| = 50, L = 30: floor(10 * 0.6 / 3) = 2 = B_min; L = 60 -> floor(1.0) -> B_min 2."""
    for p, B in ((50, 6), (275, 15), (162, 10), (20, 6), (400, 15)):
        r = oracle.sim_queue([0.0], [0], _pool_const(K=20, prompt=p), oracle.SimPolicy(early_exit=0))
        assert r["budget"][0] == B and r["chunks"][0] == B
    r = oracle.sim_queue(np.zeros(30), np.zeros(30, np.int32), _pool_const(K=20, prompt=162), oracle.SimPolicy(early_exit=0))
    assert [int(r["budget"][i]) for i in (0, 10, 15, 20, 25, 29)] == [3, 5, 6, 10, 10, 10]
    r = oracle.sim_queue(np.zeros(60), np.zeros(60, np.int32), _pool_const(K=20, prompt=50), oracle.SimPolicy(early_exit=0))
    assert r["budget"][0] == 2 and r["budget"][30] == 2 and r["budget"][59] == 6
    # the pool's chunk count caps the budget
    r = oracle.sim_queue([0.0], [0], _pool_const(K=4, prompt=275), oracle.SimPolicy(early_exit=0))
    assert r["budget"][0] == 4


def _tanh_expm1(x):
    e = math.expm1(-2.0 * abs(x))
    t = -e / (2.0 + e)
    return math.copysign(t, x)


def test_S6_ema_and_threshold_sequence_of_a_lone_request():
    """A single request alone in the system sees L = 1 at every ATP, so the EMA has the geometric
    closed form Lbar_m = 1 - 0.7^m (Lbar_0 = 0) and the threshold of ATP m is Eq. 5 at
    that value (tanh through expm1 here).  With L_target = 1 and lambda_max = 0.99 the thresholds are
    0.97417, 0.96817, 0.96321, 0.95942; confidences placed between them fix the exit chunk."""
    lam = [0.95 - 0.04 * _tanh_expm1((1 - 0.7 ** m) - 1.0) for m in (1, 2, 3, 4)]
    assert abs(lam[0] - 0.974175) < 2e-6 and abs(lam[1] - 0.968169) < 2e-6 and abs(lam[2] - 0.963206) < 2e-6
    assert abs(lam[3] - 0.959424) < 2e-6
    pol = oracle.SimPolicy(l_target=1.0, lambda_max=0.99, adaptive_budget=0, fixed_budget=4)
    for confs, chunks, exited in (
            ([0.9740, 0.9700, 0.9640, 0.5], 2, 1),     # 0.9740 <= lam1, 0.9700 > lam2
            ([0.9742, 0.5, 0.5, 0.5], 1, 1),           # 0.9742 > lam1
            ([0.9740, 0.9680, 0.9640, 0.5], 3, 1),     # 0.9680 <= lam2, 0.9640 > lam3
            ([0.9740, 0.9680, 0.9630, 0.9590], 4, 0),  # lam4 = 0.95942: never above -> budget exhausted
            ([0.9740, 0.9680, 0.9630, 0.9597], 4, 1)):
        pool = _pool_const(K=4)
        pool["conf"][0] = np.asarray(confs, np.float32)
        r = oracle.sim_queue([0.0], [0], pool, pol)
        assert (int(r["chunks"][0]), int(r["exited"][0])) == (chunks, exited), confs
    # margin = distance of the closest decision
    pool = _pool_const(K=4)
    pool["conf"][0] = np.asarray([0.9740, 0.9700, 0.9640, 0.5], np.float32)
    r = oracle.sim_queue([0.0], [0], pool, pol)
    assert abs(r["margin"][0] - abs(float(np.float32(0.9740)) - lam[0])) < 1e-12


def test_S7_load_counts_everyone_in_the_system():
    """L(t) = arrived - finished (DESIGN S1): a second request that arrives during the first one's
    second chunk raises L from 1 to 2 at that ATP.  alpha = 1 makes Lbar = L, L_target = 1.5 and
    gamma = 10 make the threshold jump from the upper clamp (L = 1) to the lower one (L = 2)."""
    pol = oracle.SimPolicy(alpha=1.0, l_target=1.5, gamma=10.0, beta=0.04, lambda_min=0.92, lambda_max=0.97,
                           adaptive_budget=0, fixed_budget=3)
    pool = _pool_const(K=3, chunk=1.0, conf=0.95, pre=0.0, conc=0.0)
    # alone: lambda = 0.97 at every ATP -> 0.95 never exits
    r = oracle.sim_queue([0.0], [0], pool, pol)
    assert r["chunks"][0] == 3 and r["exited"][0] == 0
    # second request arrives at t = 1.5: ATP 1 (t = 1) sees L = 1, ATP 2 (t = 2) sees L = 2 -> lambda 0.92 -> exit
    r = oracle.sim_queue([0.0, 1.5], [0, 0], pool, pol)
    assert r["chunks"][0] == 2 and r["exited"][0] == 1 and r["finish"][0] == 2.0
    # an arrival exactly AT the ATP time counts (arrival <= t)
    r = oracle.sim_queue([0.0, 1.0], [0, 0], pool, pol)
    assert r["chunks"][0] == 1 and r["finish"][0] == 1.0


def test_S8_summary_matches_numpy():
    pool = wl.sim_pool(seed=15)
    arr = wl.sim_arrivals_poisson(1, 1337, 0.4, seed=16)[:, 0]
    sid = wl.sim_sample_ids(1, 1337, 500, seed=17)[:, 0]
    r = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy())
    s = oracle.sim_summary(arr, r["finish"], r["chunks"], deadline=30.0)
    lat = r["finish"] - arr
    assert abs(s[0] - lat.mean()) < 1e-9
    assert s[1] == np.percentile(lat, 95, method="inverted_cdf")
    assert abs(s[2] - 1337 / (r["finish"][-1] - arr[0])) < 1e-12
    assert s[3] == (lat <= 30.0).mean() and abs(s[4] - r["chunks"].mean()) < 1e-12


def test_S9_laser_sheds_work_under_load():
    """under overload the threshold drops and budgets shrink, so LASER generates
    no more chunks than Fixed-High on any request stream, and its queue drains faster."""
    pool = wl.sim_pool(seed=18)
    arr = wl.sim_arrivals_burst(1, seed=19)[:, 0]
    sid = wl.sim_sample_ids(1, arr.shape[0], 500, seed=20)[:, 0]
    laser = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy())
    high = oracle.sim_queue(arr, sid, pool, oracle.SimPolicy(beta=0.0, adaptive_budget=0, fixed_budget=10))
    assert laser["chunks"].mean() < high["chunks"].mean()
    assert (laser["finish"] - arr).mean() < (high["finish"] - arr).mean()
    assert np.all(laser["chunks"] <= laser["budget"]) and np.all(laser["budget"] >= 2)
