"""BASELINE.json configs[1] in full: all 29 x 4 x 2 = 232 (Delta, S, order) points of the precision sweep, each held to
north_star's bounds against the CPU oracle (tests/cfg2_sweep.py: MSE within 10 %, P codes of a whole head >= 99.99 %
identical and never more than one step apart, both underflow counters, Thm 4, Eq. 7 / F* in forward order)."""
import pytest

import cfg2_sweep

pytestmark = pytest.mark.gpu


def test_cfg2_every_point():
    bad, n = [], 0
    for x in cfg2_sweep.sweep():
        n += 1
        try:
            cfg2_sweep.gate(x)
        except AssertionError as e:
            bad.append(str(e))
    assert n == 232
    assert not bad, f"{len(bad)} of {n} points outside the bounds:\n" + "\n".join(bad[:20])
