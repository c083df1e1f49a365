"""The seeded workload definitions (BASELINE.json configs and the paper's Table II schedules)."""
import math

import numpy as np

from paper_2503_14688_b200 import workloads as W


def test_baseline_configs_shapes_and_seeds():
    c = W.CONFIGS
    assert (c["ising_L64"].L, c["ising_L64"].sweeps, c["ising_L64"].r_max) == (64, 2000, 32)
    assert (c["ising_L4096"].L, c["ising_L4096"].sweeps, c["ising_L4096"].r_max) == (4096, 20000, 1024)
    assert (c["bc_L16384"].L, c["bc_L16384"].sweeps, c["bc_L16384"].r_max) == (16384, 10000, 4096)
    assert (c["ising_L2p20"].L, c["ising_L2p20"].sweeps, c["ising_L2p20"].r_max) == (1 << 20, 64, 4096)
    assert c["ising_L2p20"].state_bytes == 128 << 30
    assert c["bc_L2p15_ramp"].state_bytes == 256 << 20
    assert len({w.seed for w in c.values()}) == len(c)
    # Onsager: T_c = 2 / ln(1 + sqrt 2)
    assert abs(1.0 / W.BETA_C_ISING - 2.269185314213022) < 1e-15
    assert W.BETA_BC == 1.0 / 1.6934


def test_protocol1_and_ramp_schedules():
    w = W.CONFIGS["ising_L4096"]
    assert (w.beta_schedule(5) == W.BETA_C_ISING).all()
    r = W.CONFIGS["ising_L2p16_ramp"]
    bf = W.BETA_C_ISING / 1.01
    s = r.beta_schedule(1200)
    assert s[0] == 0.9 * bf and abs(s[999] - bf) < 1e-16 and (s[999:] == bf).all()
    assert (np.diff(s[:1000]) > 0).all()
    # a schedule is a pure function of the sweep index: slices agree
    assert np.array_equal(r.beta_schedule(50, 980), s[980:1030])


def test_paper_two_step_schedules():
    # Table II: T_1 = 1.66 / 1.24 until t_switch, then T_2
    w = W.CONFIGS["ising_L2p16_twostep"]
    s = w.beta_schedule(10, w.t_switch - 5)
    assert (s[:5] == 1.0 / 1.66).all() and (s[5:] == 1.0 / 2.27414861561203).all()
    b = W.CONFIGS["bc_L2p16_twostep"]
    s = b.beta_schedule(4, b.t_switch - 2)
    assert s.tolist() == [1 / 1.24, 1 / 1.24, 1 / 1.69661396797728, 1 / 1.69661396797728]
    # T_1 ~ 0.73 T_c
    assert abs(1.66 * W.BETA_C_ISING - 0.7315) < 1e-3


def test_measure_times():
    w = W.CONFIGS["ising_L64"]
    assert w.measure_times(20) == [0, 1, 2, 4, 8, 16, 20]
    assert w.measure_times()[-1] == 2000 and 1024 in w.measure_times()
    assert math.log2(W.CONFIGS["ising_L2p20"].spins) == 40


def _paper_values():
    import os
    vals = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        nums = []
        for tok in f[1:]:
            try:
                nums.append(float(tok))
            except ValueError:
                break
        vals[f[0]] = nums
    return vals


def test_constants_against_the_numbers_the_paper_prints():
    """tests/golden/paper_values.txt (each line cites its passage) against the workload constants
    and the constants of the estimator layer and the physics tests."""
    from paper_2503_14688_b200 import analysis
    p = _paper_values()
    assert abs(1.0 / W.BETA_C_ISING - p["Tc_ising"][0]) < 1e-15            # Onsager, 16 digits
    assert abs(2.0 / math.log(1.0 + math.sqrt(2.0)) - p["Tc_ising"][0]) < 1e-15
    assert abs(W.T_BC - p["Tc_blume_capel"][0]) < 2e-4                      # BASELINE config 3 rounds T_c to 1.6934
    assert p["E_eq_ising"][0] == -math.sqrt(2.0)
    assert analysis.OMEGA == p["omega"][0]
    i2, b2 = W.CONFIGS["ising_L2p16_twostep"], W.CONFIGS["bc_L2p16_twostep"]
    assert 1.0 / i2.beta_1 == p["ising_T1"][0] and abs(1.0 / i2.beta_f - p["ising_T2"][0]) < 1e-15
    assert i2.t_switch in [int(x) for x in p["ising_t_switch"]] and i2.sweeps == int(p["ising_t_max2"][0])
    assert abs(1.0 / b2.beta_1 - p["bc_T1"][0]) < 1e-15 and abs(1.0 / b2.beta_f - p["bc_T2"][0]) < 1e-15
    assert b2.t_switch in [int(x) for x in p["bc_t_switch"]] and b2.sweeps == int(p["bc_t_max2"][0])
    # T_1 ~ 0.73 T_c for both models
    assert abs(p["ising_T1"][0] / p["Tc_ising"][0] - 0.73) < 0.005
    assert abs(p["bc_T1"][0] / p["Tc_blume_capel"][0] - 0.73) < 0.005
    # the record: 8.7 fs per update = 114 943 updates/ns in aggregate
    assert abs(1e6 / p["time_per_update_fs"][0] - 114943) < 1
