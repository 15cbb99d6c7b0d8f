"""The frozen record-time lists follow the stated rule and the configs match BASELINE.json."""
import json
import os

import workloads


def test_record_time_rule_reproduces_frozen_lists():
    assert workloads.log_spaced_times(10_000, 40) == workloads.CONFIGS[2]["record_times"]
    assert workloads.log_spaced_times(100_000, 50) == workloads.CONFIGS[3]["record_times"]
    assert workloads.log_spaced_times(100_000, 50) == workloads.CONFIGS[5]["record_times"]
    assert workloads.log_spaced_times(1000, 20) == workloads.CONFIGS[4]["record_times"]
    assert workloads.CONFIGS[1]["record_times"] == [2 ** k for k in range(10)] + [1000]
    for key, c in workloads.CONFIGS.items():
        t = c["record_times"]
        assert all(b > a for a, b in zip(t, t[1:])) and t[0] >= 1 and t[-1] <= c["n_mcs"]
        if str(key).startswith("paper-"):
            assert t == workloads.eq7_times(c["n_mcs"])     # Eq. 7
        else:
            assert t[-1] == c["n_mcs"]


def test_eq7_sampling_times():
    """t_0 = 30, t_{i+1} = 1.05 t_i; "260 data sampling events" up to 10^7 MCS - the integer rule
    gives 270 (the first steps advance by 1 where 1.05 t rounds back to t)."""
    t = workloads.eq7_times(10**7)
    assert t[0] == 30 and t[1] == 31 and all(b > a for a, b in zip(t, t[1:]))
    assert 255 <= len(t) <= 275
    big = [x for x in t if x > 1000]
    assert all(abs(b / a - 1.05) < 0.002 for a, b in zip(big, big[1:]))


def test_configs_match_baseline_json_sizes():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with open(os.path.join(root, "BASELINE.json")) as f:
        base = json.load(f)
    assert len(base["configs"]) == 5
    c = workloads.CONFIGS
    assert (c[1]["L"], c[1]["S"], c[1]["n_mcs"], c[1]["seed"]) == (64, 16, 1000, 1)
    assert (c[2]["L"], c[2]["S"], c[2]["n_mcs"], c[2]["seed"], c[2]["p"], c[2]["q"]) == (8192, 1024, 10**4, 2, .75, .25)
    assert (c[3]["L"], c[3]["S"], c[3]["n_mcs"], c[3]["seed"], c[3]["disorder"]) == (16384, 512, 10**5, 3, (0.1, 0.5, 0.0, 0.0))
    assert (c[4]["L"], c[4]["S"], c[4]["n_mcs"], c[4]["seed"], c[4]["p"], c[4]["q"]) == (2**28, 1, 1000, 4, .9, .1)
    assert (c[5]["L"], c[5]["S"], c[5]["n_mcs"], c[5]["seed"], c[5]["turn_prob"], c[5]["turn_period"], c[5]["omega"],
            c[5]["rho0"]) == (16384, 256, 10**5, 5, 0.05, 100, 0.1, 0.3)
    assert workloads.site_updates(c[2]) == 8192 * 1024 * 10**4
    assert workloads.site_updates(c[5]) == 2 * 16384 * 256 * 10**5
