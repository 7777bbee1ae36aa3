"""Pins of the oracle's tableau (oracle/dop853_tableau.h) by the order conditions.

The paper prints no coefficient (PAPER.md:43 cites [51]; PAPER.md:129 names DOP853), so
the table is pinned by mathematics: a Runge-Kutta tableau that satisfies the conditions
below and shows slope 8 (test_oracle_step.py) is the 8th-order method whatever its source.
The header is parsed as text here: this test shares no code with the oracle.
"""
import os
import re

import numpy as np

HDR = os.path.join(os.path.dirname(__file__), "..", "oracle", "dop853_tableau.h")


def _load():
    txt = open(HDR).read()

    def arr(name):
        m = re.search(r"%s\[[^\]]*\](?:\[[^\]]*\])?\s*=\s*\{(.*?)\};" % name, txt, re.S)
        nums = re.findall(r"-?\d+\.\d+(?:e[-+]?\d+)?", m.group(1))
        return np.array([float(x) for x in nums])

    c, a, b, e5, e3 = arr("ORC_C"), arr("ORC_A").reshape(12, 12), arr("ORC_B"), arr("ORC_E5"), arr("ORC_E3")
    return c, a, b, e5, e3


def test_shapes_and_structure():
    c, a, b, e5, e3 = _load()
    assert c.shape == (12,) and b.shape == (12,) and e5.shape == (12,) and e3.shape == (12,)
    assert np.all(np.triu(a) == 0), "explicit method: A strictly lower triangular"
    assert c[0] == 0 and c[11] == 1
    assert list((a != 0).sum(1)) == [0, 1, 2, 2, 3, 3, 4, 5, 6, 7, 8, 9]
    assert list(np.nonzero(b)[0]) == [0, 5, 6, 7, 8, 9, 10, 11]


def test_row_sums():
    c, a, *_ = _load()
    assert np.max(np.abs(a.sum(1) - c)) < 1e-14


def test_quadrature_conditions_order_8():
    c, a, b, *_ = _load()
    for q in range(8):
        assert abs(b @ c ** q - 1.0 / (q + 1)) < 1e-14, q
    assert abs(b @ c ** 8 - 1.0 / 9) > 1e-6, "order is 8, not 9"


def test_second_level_conditions():
    c, a, b, *_ = _load()
    # sum_i b_i a_ij c_j^q = 1/((q+1)(q+2)), q = 0..6   (tall trees of order q+2 <= 8)
    for q in range(7):
        assert abs(b @ (a @ c ** q) - 1.0 / ((q + 1) * (q + 2))) < 1e-14, q
    # sum b_i c_i a_ij c_j^q = 1/((q+1)(q+3)), q = 0..5   (order q+3 <= 8)
    for q in range(6):
        assert abs((b * c) @ (a @ c ** q) - 1.0 / ((q + 1) * (q + 3))) < 1e-14, q
    # sum b_i a_ij a_jk c_k^q = 1/((q+1)(q+2)(q+3)), q = 0..5
    for q in range(6):
        assert abs(b @ (a @ (a @ c ** q)) - 1.0 / ((q + 1) * (q + 2) * (q + 3))) < 1e-14, q


def test_error_weights_annihilation_degrees():
    c, a, b, e5, e3 = _load()
    for q in range(5):
        assert abs(e5 @ c ** q) < 1e-14, q
    assert abs(e5 @ c ** 5) > 1e-5          # b - bhat5 sees degree-5 terms: 5th-order estimator
    for q in range(3):
        assert abs(e3 @ c ** q) < 1e-14, q
    assert abs(e3 @ c ** 3) > 1e-3          # 3rd-order estimator
