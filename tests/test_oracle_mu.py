"""Pins for oracle step 7: log-log mu(E) interpolation."""
import numpy as np


def test_power_law_is_reproduced_exactly(O):
    E = np.exp(np.linspace(np.log(10), np.log(150), 1000))
    tab = {"E": E, "mu": 37.0 * (E / 30.0) ** -2.9}
    for Eq in np.random.default_rng(0).uniform(10, 150, 200):
        assert abs(O.mu(tab, Eq) / (37.0 * (Eq / 30.0) ** -2.9) - 1) < 1e-13
    # end segments extrapolate (R11)
    assert abs(O.mu(tab, 8.0) / (37.0 * (8.0 / 30.0) ** -2.9) - 1) < 1e-13
    assert abs(O.mu(tab, 200.0) / (37.0 * (200.0 / 30.0) ** -2.9) - 1) < 1e-13


def test_exact_at_knots_and_geometric_mean_midpoint(O, W):
    tab = W.mu_table(np.random.default_rng(3))
    for j in (0, 1, 17, 500, 998, 999):
        assert abs(O.mu(tab, tab["E"][j]) / tab["mu"][j] - 1) < 1e-13
    # at the geometric mean of two knots log-log interpolation gives the geometric mean of the values
    j = 300
    Em = np.sqrt(tab["E"][j] * tab["E"][j + 1])
    assert abs(O.mu(tab, Em) / np.sqrt(tab["mu"][j] * tab["mu"][j + 1]) - 1) < 1e-13


def test_edge_jump(O, W):
    tab = W.mu_table(np.random.default_rng(5))
    ratio = tab["mu"][1:] / tab["mu"][:-1]
    j = int(np.argmax(ratio))
    assert ratio[j] > 2.9                                        # a jump of x3..x6
    Ee = 0.5 * (tab["E"][j] + tab["E"][j + 1])
    below, above = O.mu(tab, Ee * (1 - 2e-6)), O.mu(tab, Ee * (1 + 2e-6))
    assert abs(above / below / ratio[j] - 1) < 1e-4
    assert O.mu(tab, Ee * (1 - 1e-3)) > O.mu(tab, Ee * (1 - 2e-6))  # decreasing below the edge


def test_vacuum_is_zero(O, W):
    box = W.solids([W.solid_box((1e-2, 1e-2, 1e-2), material=0, priority=0, T=(0, 0, 0.5))])
    rc, st, _ = O.apply(box, [0, 0, 0, 0, 0, 1, 20.0, 0.8], materials=[None])
    assert rc == 1 and st[7] == 0.8
