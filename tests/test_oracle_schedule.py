"""Pins of the Eq.17 learning-rate schedule (paper P:117-126): the oracle's restatement against what the formula
fixes, and the library's host function gnep_lr_schedule (no GPU needed: pure host arithmetic) against the oracle."""
import numpy as np
import pytest

from oracle import gnep_oracle as orc

A, B, NW, NT = 1e-3, 1e-5, 40, 400          # lr_start, lr_stop, warm-up steps, total steps


def test_end_points_and_special_values():
    assert orc.lr_schedule(0, NW, NT, A, B) == B                               # starts at the minimum
    assert orc.lr_schedule(NW, NW, NT, A, B) == pytest.approx(A, rel=1e-15)    # peak at the end of the warm-up
    assert orc.lr_schedule(NT, NW, NT, A, B) == pytest.approx(B, rel=1e-12)    # back at the minimum
    mid = NW + (NT - NW) // 2
    assert orc.lr_schedule(mid, NW, NT, A, B) == pytest.approx(0.5 * (A + B), rel=1e-12)   # cos(pi/2) = 0
    q = NW + (NT - NW) // 3                                                    # cos(pi/3) = 1/2
    assert orc.lr_schedule(q, NW, NT, A, B) == pytest.approx(B + 0.75 * (A - B), rel=1e-12)


def test_warmup_is_linear_and_decay_is_monotone():
    w = np.array([orc.lr_schedule(s, NW, NT, A, B) for s in range(NW + 1)])
    np.testing.assert_allclose(np.diff(w), (A - B) / NW, rtol=1e-9)
    d = np.array([orc.lr_schedule(s, NW, NT, A, B) for s in range(NW, NT + 1)])
    assert np.all(np.diff(d) < 0) and np.all(d >= B - 1e-18) and np.all(d <= A + 1e-18)
    # the two branches meet: continuity at s = NW
    assert abs(w[-1] - d[0]) < 1e-18
    # no warm-up at all: pure cosine from lr_start
    assert orc.lr_schedule(0, 0, NT, A, B) == pytest.approx(A, rel=1e-15)


def test_library_host_function_matches():
    from paper_2507_00528_b200 import GnepError, lr_schedule
    for nw, nt in ((NW, NT), (0, 7), (5, 5), (3, 10)):
        for s in list(range(0, nt + 1)) + [-3, nt + 9]:
            assert lr_schedule(s, nw, nt, A, B) == pytest.approx(orc.lr_schedule(s, nw, nt, A, B), rel=1e-14, abs=1e-20)
    for bad in ((0, 5, 3), (0, -1, 3), (0, 0, 0)):
        with pytest.raises(GnepError):
            lr_schedule(bad[0], bad[1], bad[2], A, B)
