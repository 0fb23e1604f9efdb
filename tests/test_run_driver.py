"""Host-side helpers of the run driver (time grid, effective exponents of Eq. (8))."""
import math

import pytest

from paper_1705_01022_b200 import run


def test_log_grid_is_sorted_unique_and_ends_at_t_max():
    g = run.log_grid(10_000, 8)
    assert g[0] == 1 and g[-1] == 10_000 and g == sorted(set(g))
    assert all(b > a for a, b in zip(g, g[1:]))
    assert 30 <= len(g) <= 40                                  # ~8 points per decade over 4 decades
    assert run.log_grid(1, 8) == [1]


def test_effective_exponent_recovers_a_power_law():
    # E = 3 t^0.4828 (2 beta with beta = 0.2414) -> e_eff = 0.4828 between any two points
    f = lambda t: 3.0 * t ** 0.4828
    for t0, t1 in ((10, 20), (100, 1000), (7, 5000)):
        assert run.eff_exponent(f(t1), t1, f(t0), t0) == pytest.approx(0.4828, rel=1e-12)
    assert run.eff_exponent(1.0, 10, 0.0, 5) is None and run.eff_exponent(1.0, 5, 1.0, 5) is None
    assert math.isclose(run.eff_exponent(0.5, 4, 1.0, 2), -1.0)


def test_ensemble_mean_and_standard_error():
    runs = [[{"t": 1, "w2": 1.0, "mean_h": 0.5}, {"t": 10, "w2": 4.0, "mean_h": 5.0}],
            [{"t": 1, "w2": 3.0, "mean_h": 0.5}, {"t": 10, "w2": 6.0, "mean_h": 7.0}]]
    e = run.ensemble_mean(runs)
    assert [r["t"] for r in e] == [1, 10] and e[0]["n"] == 2
    assert e[0]["w2"] == 2.0 and e[0]["w2_sem"] == pytest.approx(1.0)        # sqrt(((1)^2+(1)^2)/(2*1))
    assert e[1]["w2"] == 5.0 and e[1]["mean_h_sem"] == pytest.approx(1.0)
    assert e[1]["beta_eff"] == pytest.approx(math.log(5.0 / 2.0) / math.log(10.0) / 2)
    # propagated 1-sigma error: sqrt((1/5)^2 + (1/2)^2) / ln 10 / 2, and the spread of the per-run exponents
    assert e[1]["beta_eff_err"] == pytest.approx(math.sqrt(0.2 ** 2 + 0.5 ** 2) / math.log(10.0) / 2)
    b = [math.log(4.0) / math.log(10.0) / 2, math.log(2.0) / math.log(10.0) / 2]
    assert e[1]["beta_eff_sem"] == pytest.approx(abs(b[0] - b[1]) / 2)
    assert "c_h" not in e[0]


def test_aging_exponent_and_its_error_use_t_over_s():
    # C_h = 7 (t/s)^(-1.21) (lambda_h/z of PAPER.md:100-104 is about 1.21 for KPZ): recovered between any two points
    s = 100.0
    f = lambda t: 7.0 * (t / s) ** -1.21
    runs = [[{"t": 200.0, "w2": 1.0, "c_h": f(200.0) * k}, {"t": 400.0, "w2": 2.0, "c_h": f(400.0) * k}] for k in (0.9, 1.1)]
    e = run.ensemble_mean(runs, snap_t=s)
    assert e[1]["lambda_h_over_z_eff"] == pytest.approx(1.21)
    rel = 0.1 / math.sqrt(2) * math.sqrt(2)          # each point: values 0.9x and 1.1x -> sem = 0.1 x
    assert e[1]["lambda_h_over_z_eff_err"] == pytest.approx(math.sqrt(2) * rel / math.log(2.0))
    assert run.eff_exponent_err(1.0, 0.1, 10, 0.0, 0.1, 5) is None


def test_member_groups_partition_the_ensemble():
    # groups are contiguous, disjoint and cover every member; one member or a large lattice stays in one group
    for n, L, g in ((1, 1024, 0), (2, 1024, 0), (32, 1024, 0), (33, 1024, 2), (7, 1024, 4), (8, 65536, 0), (5, 1024, 9)):
        groups = run.member_groups(n, L, g)
        assert [i for grp in groups for i in grp] == list(range(n))
        assert all(grp for grp in groups)
    assert len(run.member_groups(1, 1024)) == 1 and len(run.member_groups(32, 1024)) == 1 and len(run.member_groups(32, 1024, 2)) == 2
    assert len(run.member_groups(8, 65536)) == 1 and len(run.member_groups(5, 1024, 9)) == 5
    assert [len(g) for g in run.member_groups(33, 1024, 2)] == [17, 16]
