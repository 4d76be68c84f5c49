"""CPU: the bookkeeping of tests/parity.py that decides whether a stop block that differs from the oracle's on a FRAGILE
group is legitimate (north_star: such groups are 'reported separately')."""
import numpy as np

from parity import reachable_stops, FRAGILE_REL


def trace(ds, dd=None):
    ds = np.asarray(ds, float)[:, None]
    dd = np.zeros_like(ds) if dd is None else np.asarray(dd, float)[:, None]
    return ds, dd


def test_nothing_near_the_threshold_gives_exactly_the_sequential_stop():
    tau, phi = 1e-2, 1e-3
    ds, dd = trace([1, .5, .1, 5e-3, 4e-3, 3e-3, 2e-3, 1e-3, 9e-4])
    assert reachable_stops(ds, dd, tau, phi, 3) == {6}           # stable from t = 4: 4, 5, 6
    assert reachable_stops(ds, dd, tau, phi, 7) == {9}           # never reaches 7 in a row: T
    assert reachable_stops(ds, dd, 0.0, phi, 1) == {9}           # tau = 0: never stable


def test_a_value_on_the_threshold_may_go_either_way():
    tau, phi = 1e-2, 1e-3
    near = tau * (1 + 0.5 * FRAGILE_REL)
    ds, dd = trace([1, near, 5e-3, 5e-3, 5e-3, 5e-3])
    assert reachable_stops(ds, dd, tau, phi, 3) == {4, 5}        # run starts at t = 2 (if it passes) or at t = 3
    ds, dd = trace([1, 5e-3, 5e-3, near, 5e-3, 5e-3, 5e-3, 1, 1])
    assert reachable_stops(ds, dd, tau, phi, 3) == {4, 7}        # fires at 4, or the run is broken and restarts
    ds, dd = trace([1, 5e-3, tau * (1 + 3 * FRAGILE_REL), 5e-3, 5e-3, 5e-3])
    assert reachable_stops(ds, dd, tau, phi, 3) == {6}           # outside the band: a sure 'not stable'


def test_direction_and_heads_combine_with_and():
    tau, phi = 1e-2, 1e-3
    ds = np.full((5, 2), 1e-3); dd = np.zeros((5, 2))
    dd[2, 1] = phi * (1 - 0.5 * FRAGILE_REL)                      # head 1 sits on phi at t = 3
    assert reachable_stops(ds, dd, tau, phi, 3) == {3, 5}         # (no zero-norm first step in this synthetic trace)
    dd[2, 1] = 1.0
    assert reachable_stops(ds, dd, tau, phi, 2) == {2}
    assert reachable_stops(ds, dd, tau, float("inf"), 5) == {5}
