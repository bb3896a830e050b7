"""Grid helper / period post-processing against the values the paper prints (tests/golden/table2_frequency_grid.txt:
Table 2, and the frequency <-> period pairs of PAPER.md:L236, L240, L289)."""
import math
import os

import numpy as np
import pytest

from paper_2105_04006_b200 import grid

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "table2_frequency_grid.txt")


def _rows():
    out = []
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append(line.split())
    return out


def test_table2_n_freq_from_printed_ranges():
    rows = [r for r in _rows() if r[0] in ("single_object", "batch")]
    assert len(rows) == 2
    for name, f_min, f_max, df, n_f in rows:
        assert grid.n_freq_for(float(f_min), float(f_max), float(df)) == int(n_f), name
        # the same grid through the cyclic API: N_f does not depend on the unit
        assert grid.n_freq_for(grid.angular_to_cyclic(float(f_min)), grid.angular_to_cyclic(float(f_max)),
                               grid.angular_to_cyclic(float(df))) == int(n_f), name


def test_table2_delta_f_is_the_richards_rule_for_a_120_day_window():
    # delta_f = 0.2 pi / T_max.  Table 2's 5.237e-3 rad/day is a window of 119.98 d (Fig. 1's ~120 d baseline);
    # the angular and cyclic forms of the rule agree.
    for name, _, _, df, _ in [r for r in _rows() if r[0] in ("single_object", "batch")]:
        t_max = 0.2 * math.pi / float(df)
        assert 119.9 < t_max < 120.1
        assert grid.delta_f(t_max, angular=True) == pytest.approx(float(df), rel=1e-12)
        assert grid.cyclic_to_angular(grid.delta_f(t_max)) == pytest.approx(float(df), rel=1e-12)


def test_printed_frequency_period_pairs():
    for _, f, p_lc, p_rot in [r for r in _rows() if r[0] == "period"]:
        p_hours = 24.0 * float(grid.light_curve_period(float(f), angular=True))
        assert p_hours == pytest.approx(float(p_lc), rel=2e-3)          # the paper prints f to 4 significant digits
        assert 24.0 * float(grid.rotation_period(grid.light_curve_period(float(f), angular=True))) == pytest.approx(float(p_rot), rel=2e-3)
        assert float(grid.light_curve_period(grid.angular_to_cyclic(float(f)))) == pytest.approx(p_hours / 24.0, rel=1e-12)


def test_observing_window_and_practical_grid():
    offsets = np.array([0, 3, 3, 7])
    t = np.array([10.0, 12.0, 70.0, 5.0, 125.0, 6.0, 9.0])
    assert grid.observing_window(offsets, t) == 120.0          # max(60, -, 120); the empty object is skipped
    f_min, f_max, n_freq = grid.practical_grid(offsets, t, 0.5, 24.0)
    assert (f_min, f_max) == (0.5, 24.0) and n_freq == round(23.5 / (0.1 / 120.0))
    with pytest.raises(ValueError):
        grid.delta_f(0.0)
    with pytest.raises(ValueError):
        grid.n_freq_for(2.0, 1.0, 0.1)
